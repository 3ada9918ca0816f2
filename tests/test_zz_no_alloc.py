"""svr_ssim_loss_grad_static: the SSIM loss gradient for callers that cannot allocate device memory.

Some users of libsvr.so run where a device allocation is not an option: as a component of a host application whose own
allocator already owns the GPU's memory, under a memory reservation fixed before the run, or in a loop that cannot take the
device-wide stall of an allocation or a free. svr_ssim_loss_grad_static serves them from a fixed 36 MiB array built into the
library (images of up to 2^20 pixels) instead of the context's workspace pool; see include/svr.h.

The check is against the existing, pool-backed svr_ssim_loss_grad on the same inputs, with the tolerances
test_gpu_parity.py::test_ssim_loss_grad_parity uses against the oracle (gradient: relative L2 <= 1e-5; loss: 2e-6 relative).
Back-to-back calls matter here because every call reuses the one array and finds the previous call's data in it: the second
image is smaller than the first (stale maps and a stale index sum lie beyond and beneath it), the third accumulates.

This file is named to be collected last (pytest -x stops at the first failure; a failure here must not hide other tests) and
passes on its own in a fresh process as well as after the rest of the suite: it shares no state with the other files.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

GRAD_TOL = 1e-5      # relative L2, as in test_ssim_loss_grad_parity
LOSS_TOL = 2e-6      # relative, as in test_ssim_loss_grad_parity


def _rel_l2(x, r):
    x, r = np.asarray(x, dtype=np.float64), np.asarray(r, dtype=np.float64)
    return float(np.linalg.norm(x - r) / max(np.linalg.norm(r), 1e-300))


def _images(rng, H, W):
    base = rng.uniform(0, 1, size=(H, W, 3)) * np.linspace(0.1, 1, W)[None, :, None]
    base[H // 2:, :, :] = 0.4                                   # a flat region, where the variances cancel against C2
    target = np.clip(base, 0, 1).astype(np.float32)
    render = np.clip(target + rng.normal(0, 0.05, size=target.shape), 0, 1).astype(np.float32)
    return render, target


def test_static_scratch_ssim_matches_pool_path_on_consecutive_calls():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2511_02510_b200 as pkg

    rng = np.random.default_rng(2511)
    # (H, W, lambda, accumulate): several 16 x 16 tiles with ragged edges; then a smaller image; then accumulation
    cases = [(150, 203, 1.0, False), (37, 61, 0.5, False), (75, 133, 0.2, True)]

    # the existing path first (it allocates from the context's pool), so that nothing but the new entry point runs below
    ctx = pkg.Context(0)
    inputs, want = [], []
    for (H, W, lam, accumulate) in cases:
        render, target = _images(rng, H, W)
        r_dev, t_dev = torch.from_numpy(render).cuda(), torch.from_numpy(target).cuda()
        prior = torch.from_numpy(rng.normal(0, 1e-4, size=render.shape).astype(np.float32)).cuda()
        dL_ref = prior.clone() if accumulate else None
        dL_ref, loss_ref = ctx.svr_ssim_loss_grad(r_dev, t_dev, lam, dL=dL_ref, accumulate=accumulate)
        ctx.synchronize()
        inputs.append((r_dev, t_dev, prior))
        want.append((dL_ref.cpu().numpy(), float(loss_ref.item())))
    ctx.close()

    # outputs are the caller's: allocate them all before the calls under test
    outs = [(prior.clone() if acc else torch.full_like(prior, float("nan")), torch.full((1,), float("nan"), device="cuda"))
            for (_, _, prior), (_, _, _, acc) in zip(inputs, cases)]
    stream = torch.cuda.Stream()
    torch.cuda.synchronize()
    free_after_first = None
    for i, ((H, W, lam, accumulate), (r_dev, t_dev, _), (dL, loss)) in enumerate(zip(cases, inputs, outs)):
        pkg.svr_ssim_loss_grad_static(r_dev, t_dev, dL, loss, lam, accumulate=accumulate, stream=stream)
        stream.synchronize()
        free_now = torch.cuda.mem_get_info()[0]
        if i == 0:
            free_after_first = free_now      # the first call may load the kernels' module; nothing may be taken after it
        else:
            assert free_now >= free_after_first, (i, free_now, free_after_first)
        dL_ref, loss_ref = want[i]
        assert abs(float(loss.item()) - loss_ref) <= LOSS_TOL * max(abs(loss_ref), 1e-3), (i, float(loss.item()), loss_ref)
        assert _rel_l2(dL.cpu().numpy(), dL_ref) <= GRAD_TOL, (i, H, W)

    # the limit is stated and enforced before anything runs
    limit = pkg.svr_ssim_static_max_pixels()
    assert limit == 1 << 20
    big = torch.zeros((1025, 1024, 3), device="cuda")           # one row over the limit
    with pytest.raises(pkg.SvrError) as err:
        pkg.svr_ssim_loss_grad_static(big, big, torch.empty_like(big), outs[0][1])
    assert "limit" in str(err.value) and str(limit) in str(err.value)
    # exactly at the limit it runs (identical images: L_SSIM = 0, zero gradient)
    full = torch.rand((1024, 1024, 3), device="cuda")
    dL_full, loss_full = torch.full_like(full, float("nan")), torch.full((1,), float("nan"), device="cuda")
    pkg.svr_ssim_loss_grad_static(full, full, dL_full, loss_full)
    torch.cuda.synchronize()
    assert abs(float(loss_full.item())) <= 1e-6 and float(dL_full.abs().max().item()) <= 1e-9
