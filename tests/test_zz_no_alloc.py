"""sfft_mask_fill_static: the crowded-field mask/fill for callers that cannot allocate on the device.

Some users of the library run where a cudaMalloc is off the table: all device memory already belongs to one pool that
was sized at start-up (a later cudaMalloc fails or escapes the pool's bookkeeping), or the call sits in a loop that may
not stall (cudaMalloc and cudaFree synchronise the whole device).  For them the library has one entry point that takes
the input and output images and nothing else; its scratch is an array built into the library (good for frames of up to
4096 x 4096 pixels) instead of the plan's workspace.

The check: on the same seeded, saturated pair the new entry point must give what the plan-based sfft_mask_fill gives
(mask bit for bit, filled images within the 1e-12 * saturation level the mask/fill parity tests use), twice in a row
on frames of different sizes -- the second call finds the first call's leftovers in the shared scratch and must not
be disturbed by them -- and a frame beyond the limit must be refused with a message that names the limit.

This file is named so that pytest collects it last: a failure here must not hide the parity tests under `-x`.  It
depends on no state left by other tests (and leaves none): it passes alone in a fresh process and after the others.
"""
import numpy as np
import pytest

import synth
from paper_2109_09334_b200 import binding as B

SAT = 3000.0


def _saturated_pair(H, W, seed):
    """A seeded star field with its brightest stars clipped into saturated blobs with bleed columns (some of them
    crossing the frame edge, so the wrap-around of the windows is exercised)."""
    p = synth.make_pair(1, H=H, W=W)
    rng = np.random.default_rng(seed)
    R, S = p.R.copy(), p.S.copy()
    for q in np.argsort(R.ravel())[-12:]:
        x, y = divmod(int(q), W)
        for dx in range(-int(rng.integers(2, 6)), 6):
            R[(x + dx) % H, y] = SAT * 1.3
            S[(x + dx) % H, (y + 1) % W] = SAT * 1.1
    R[0, 0] = S[H - 1, W - 1] = SAT * 2
    return R, S


@pytest.mark.gpu
def test_mask_fill_static_matches_plan_path_on_two_calls_in_a_row(cuda_device):
    import torch
    # second frame smaller and not a power of two: the scratch still holds the flags and sums of the first call
    for call, (H, W, rd, rb) in enumerate([(192, 256, 2, 6), (96, 130, 3, 9)]):
        R, S = _saturated_pair(H, W, seed=call)
        dR, dS = torch.from_numpy(R).cuda(), torch.from_numpy(S).cuda()
        # the caller of the no-allocation entry point brings its outputs (poisoned here so that unwritten pixels show)
        Rm = torch.full_like(dR, float("nan"))
        Sm = torch.full_like(dS, float("nan"))
        mask = torch.full((H, W), 7, dtype=torch.uint8, device=cuda_device)
        B.mask_fill_static(dR, dS, SAT, SAT, rd, rb, Rm, Sm, mask)
        torch.cuda.synchronize()
        # existing path: a plan with a lent workspace
        plan = B.Plan(H, W, 7, 1, 1, "poly")
        Rm0, Sm0, mask0 = plan.mask_fill(dR, dS, SAT, SAT, rd, rb)
        torch.cuda.synchronize()        # (sfft_plan_status reports on the last solve; none was run here)
        plan.close()
        assert int(mask0.sum()) > 0, "the input must have saturated pixels for the comparison to mean anything"
        assert torch.equal(mask, mask0.reshape(H, W)), f"call {call}: masks differ"
        assert float((Rm - Rm0.reshape(H, W)).abs().max()) <= 1e-12 * SAT, f"call {call}: filled reference differs"
        assert float((Sm - Sm0.reshape(H, W)).abs().max()) <= 1e-12 * SAT, f"call {call}: filled science image differs"
        assert torch.equal(Rm[mask == 0], dR[mask == 0]) and torch.equal(Sm[mask == 0], dS[mask == 0])


@pytest.mark.gpu
def test_mask_fill_static_refuses_frames_beyond_its_scratch(cuda_device):
    import torch
    small = torch.zeros((32, 64), dtype=torch.float64, device=cuda_device)
    m = torch.zeros((32, 64), dtype=torch.uint8, device=cuda_device)
    ptrs = (small.data_ptr(), small.data_ptr())
    outs = (small.data_ptr(), small.data_ptr(), m.data_ptr())
    # 4096 x 4097 pixels: one row over the limit; refused before any pointer is touched
    st = B.sfft_mask_fill_static(*ptrs, 4097, 4096, SAT, SAT, 1, 2, *outs)
    assert st == B.SFFT_ERR_INVALID_ARG
    msg = B.sfft_static_last_error()
    assert str(B.SFFT_STATIC_MAX_PIXELS) in msg and "4097" in msg
    assert B.sfft_mask_fill_static(*ptrs, 32, 20000, SAT, SAT, 1, 2, *outs) == B.SFFT_ERR_INVALID_ARG
    assert B.sfft_mask_fill_static(*ptrs, 32, 64, SAT, SAT, 1, 0, *outs) == B.SFFT_ERR_INVALID_ARG
    assert B.sfft_mask_fill_static(0, small.data_ptr(), 32, 64, SAT, SAT, 1, 2, *outs) == B.SFFT_ERR_INVALID_ARG


@pytest.mark.gpu
def test_mask_fill_static_at_its_largest_frame(cuda_device):
    """4096 x 4096, the largest frame the built-in scratch holds (every byte of it is used), against the plan path."""
    import torch
    H = W = 4096
    g = torch.Generator(device=cuda_device).manual_seed(20210909)
    dR = 100.0 + 10.0 * torch.randn((H, W), dtype=torch.float64, device=cuda_device, generator=g)
    dS = 100.0 + 10.0 * torch.randn((H, W), dtype=torch.float64, device=cuda_device, generator=g)
    hot = torch.randint(0, H * W, (300,), device=cuda_device, generator=g)
    dR.view(-1)[hot] = SAT * 1.5
    dS.view(-1)[(hot[:100] + 1) % (H * W)] = SAT * 1.2
    dR[H - 1, W - 1] = dS[0, 0] = SAT * 2                      # last and first byte of the flag array matter
    Rm, Sm = torch.empty_like(dR), torch.empty_like(dS)
    mask = torch.empty((H, W), dtype=torch.uint8, device=cuda_device)
    B.mask_fill_static(dR, dS, SAT, SAT, 2, 5, Rm, Sm, mask)
    plan = B.Plan(H, W, 7, 1, 1, "poly")
    Rm0, Sm0, mask0 = plan.mask_fill(dR, dS, SAT, SAT, 2, 5)
    torch.cuda.synchronize()
    plan.close()
    assert int(mask0.sum()) >= 300 * 25 // 2
    assert torch.equal(mask, mask0) and bool(mask[H - 1, W - 1]) and bool(mask[0, 0])
    assert float((Rm - Rm0).abs().max()) <= 1e-12 * SAT and float((Sm - Sm0).abs().max()) <= 1e-12 * SAT


@pytest.mark.gpu
def test_mask_fill_static_odd_width_and_unaligned_images(cuda_device):
    """Frames the plan path does not take (odd W) and images that start on an 8-byte but not a 16-byte boundary go
    through the one-pixel-per-thread kernels: checked against the CPU oracle (mask bit for bit, fills to 1e-12 * sat),
    and the unaligned call against the aligned one on the same pixels."""
    import torch
    import oracle
    H, W, rd, rb = 97, 131, 2, 5
    R, S = _saturated_pair(H, W, seed=5)
    Rmo, Smo, mo = oracle.mask_fill(R, S, SAT, SAT, rd, rb)
    dR, dS = torch.from_numpy(R).cuda(), torch.from_numpy(S).cuda()
    Rm, Sm = torch.empty_like(dR), torch.empty_like(dS)
    mask = torch.empty((H, W), dtype=torch.uint8, device=cuda_device)
    B.mask_fill_static(dR, dS, SAT, SAT, rd, rb, Rm, Sm, mask)
    assert mo.sum() > 0 and np.array_equal(mask.cpu().numpy(), mo)
    assert np.max(np.abs(Rm.cpu().numpy() - Rmo)) <= 1e-12 * SAT and np.max(np.abs(Sm.cpu().numpy() - Smo)) <= 1e-12 * SAT
    # even width, but every image shifted by one double (and the mask by one byte) inside a larger buffer
    H, W = 64, 130
    R, S = _saturated_pair(H, W, seed=6)
    Rmo, Smo, mo = oracle.mask_fill(R, S, SAT, SAT, rd, rb)
    bufs = [torch.zeros(H * W + 1, dtype=torch.float64, device=cuda_device) for _ in range(4)]
    mbuf = torch.zeros(H * W + 1, dtype=torch.uint8, device=cuda_device)
    uR, uS, uRm, uSm = [b[1:].view(H, W) for b in bufs]
    umask = mbuf[1:].view(H, W)
    assert uR.data_ptr() % 16 == 8 and umask.data_ptr() % 2 == 1
    uR.copy_(torch.from_numpy(R)); uS.copy_(torch.from_numpy(S))
    B.mask_fill_static(uR, uS, SAT, SAT, rd, rb, uRm, uSm, umask)
    aR, aS = uR.clone(), uS.clone()
    aRm, aSm, amask = torch.empty_like(aR), torch.empty_like(aS), torch.empty((H, W), dtype=torch.uint8, device=cuda_device)
    B.mask_fill_static(aR, aS, SAT, SAT, rd, rb, aRm, aSm, amask)
    for m_, r_, s_ in ((umask, uRm, uSm), (amask, aRm, aSm)):
        assert np.array_equal(m_.cpu().numpy(), mo)
        assert np.max(np.abs(r_.cpu().numpy() - Rmo)) <= 1e-12 * SAT and np.max(np.abs(s_.cpu().numpy() - Smo)) <= 1e-12 * SAT
