"""The no-allocation entry point mred_estimate_shifts_static (include/mred.h): the scratch of the estimate kernels lives
in a static device array inside libmred.so, so the call needs no workspace and calls no cudaMalloc.  Its output must
equal the existing path's (mred_estimate_shifts_peak with a caller's workspace: same kernels, so bit for bit, which is
inside the 1e-3 px bar of the parity tests) on two calls in a row -- the second call finds the first call's contents in
the shared array -- and sizes beyond the array are refused.  Collected last (file name), so that a failure here cannot
hide another test under `pytest -x`; it passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu


def _star_frames(rng, offs, h, w, pad=32):
    H, W = h + 2 * pad, w + 2 * pad
    yy, xx = np.mgrid[0:H, 0:W]
    big = rng.normal(1000.0, 10.0, size=(H, W))
    for _ in range(40):
        x, y, a = rng.uniform(0, W), rng.uniform(0, H), np.exp(rng.uniform(np.log(200), np.log(20000)))
        big += a * np.exp(-0.5 * ((xx - x) ** 2 + (yy - y) ** 2) / 1.274 ** 2)
    return np.stack([big[pad - b:pad - b + h, pad - a:pad - a + w] for a, b in offs]).astype(np.float32)


def test_estimate_shifts_static_matches_workspace_path_twice():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2008_11486_b200 import binding as mred
    mred.lib()
    rng = np.random.default_rng(77)
    # two different stacks (different n, shape, reference, mask) so that the second call cannot pass on leftovers
    cases = [
        dict(offs=[(0, 0), (5, -3), (-17, 11), (1, 0), (20, -20), (-2, 7)], h=97, w=131, ref=0, lag=21, mask=True, peak=0),
        dict(offs=[(3, 1), (0, 0), (-6, 9)], h=200, w=260, ref=1, lag=16, mask=False, peak=1),
    ]
    for rep in range(2):                       # the whole sequence twice: four calls on the one shared array
        for c in cases:
            fr = _star_frames(rng, c["offs"], c["h"], c["w"])
            bad = None
            if c["mask"]:
                b = np.zeros((c["h"], c["w"]), np.uint8)
                b[:, 13] = 1
                b[5, :] = 1
                fr[:, :, 13] += 30000.0
                bad = torch.from_numpy(b).cuda()
            d = torch.from_numpy(fr).cuda()
            n = fr.shape[0]
            ish_ref, sh_ref = mred.estimate_shifts(d, c["ref"], c["lag"], badmask=bad, peak=c["peak"])
            ish = torch.full((n, 2), -999, dtype=torch.int32, device="cuda")
            sh = torch.full((n, 2), -999.0, dtype=torch.float64, device="cuda")
            torch.cuda.synchronize()
            before = torch.cuda.memory_allocated()
            mred.estimate_shifts_static(d, ish, sh, c["ref"], c["lag"], badmask=bad, peak=c["peak"])
            assert torch.cuda.memory_allocated() == before          # the binding allocates nothing either
            torch.cuda.synchronize()
            assert np.array_equal(ish.cpu().numpy(), ish_ref.cpu().numpy())
            assert np.max(np.abs(sh.cpu().numpy() - sh_ref.cpu().numpy())) <= 1e-3      # the parity tests' bar for shifts
            assert np.array_equal(sh.cpu().numpy(), sh_ref.cpu().numpy())               # same kernels: in fact identical
            got = ish.cpu().numpy()                                                     # and not a trivial agreement:
            assert np.all(got[c["ref"]] == 0) and np.count_nonzero(got) >= n - 1        # the frames were shifted


def test_estimate_shifts_static_refuses_sizes_beyond_its_scratch():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2008_11486_b200 import binding as mred
    g = mred.Geom(0, 0, 0, 0, 0, 0, 2048, 2048)
    n = 64
    assert mred.workspace_bytes(mred.CALL_ESTIMATE_SHIFTS, g, n) > mred.STATIC_SCRATCH_BYTES
    d = torch.zeros((n, 2048, 2048), dtype=torch.float32, device="cuda")
    ish = torch.zeros((n, 2), dtype=torch.int32, device="cuda")
    sh = torch.zeros((n, 2), dtype=torch.float64, device="cuda")
    with pytest.raises(mred.MredError, match="static scratch"):
        mred.estimate_shifts_static(d, ish, sh, 0, 8)
    # the largest 1074 x 1024 configuration (64 frames, config 4) fits
    assert mred.workspace_bytes(mred.CALL_ESTIMATE_SHIFTS, mred.Geom(0, 0, 0, 0, 0, 0, 1024, 1024), 64) <= mred.STATIC_SCRATCH_BYTES
