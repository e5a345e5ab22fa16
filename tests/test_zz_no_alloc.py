"""The allocation-free entry point sharp_fft2_noalloc (include/sharp_b200.h): batched 256 x 256 unitary DFT with the
kernel's transposition scratch in a static device array of the library, for callers that cannot call cudaMalloc.

Checked against the existing path (sharp_op_fft2 on a bound plan, whose scratch lives in the caller's workspace) on two
calls in a row, within the operator tolerance of the other GPU tests, and against the oracle on sampled frames.  This
file sorts last on purpose (pytest -x): it must pass alone in a fresh process and after all the others.
"""
import numpy as np
import pytest

import paper_1602_01448_b200 as sharp

pytestmark = pytest.mark.gpu

OP_TOL = 1e-5
M = 256


def rel(a, b):
    a = np.asarray(a); b = np.asarray(b)
    return float(np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300))


def _frames(K, seed):
    import torch
    g = torch.Generator(device="cpu").manual_seed(seed)
    re = torch.randn((K, M, M), generator=g)
    im = torch.randn((K, M, M), generator=g)
    return torch.complex(re, im).to(torch.complex64).cuda()


def test_noalloc_fft2_matches_the_existing_path_on_two_calls_in_a_row(oracle):
    import torch
    K = 40                                                     # 16 clusters in flight: 2.5 rounds, ragged last one
    pos = np.array([[8 * (i % 5), 8 * (i // 5)] for i in range(K)], np.int32)
    rec = sharp.Reconstruction(M, pos, (M + 64, M + 64))      # the existing path: plan + caller workspace
    got1 = torch.empty((K, M, M), dtype=torch.complex64, device="cuda")
    got2 = torch.empty_like(got1)
    out = torch.empty_like(got1)
    f1, f2 = _frames(K, 1), _frames(K, 2)
    sharp.fft2_noalloc(f1[:1].contiguous(), out[:1], -1)      # first use on this device: symbol addresses, module load
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    # first call: forward transform; second call, directly after it on the same stream: other data, adjoint transform
    # (the static scratch still holds the first call's contents)
    sharp.fft2_noalloc(f1, got1, -1)
    sharp.fft2_noalloc(f2, got2, +1)
    torch.cuda.synchronize()
    # driver-level free memory: a cudaMalloc inside the calls would take at least one 2 MiB granule
    assert free0 - torch.cuda.mem_get_info()[0] < (2 << 20)
    want1 = rec.op_fft2(f1, -1)
    want2 = rec.op_fft2(f2, +1)
    assert rel(got1.cpu().numpy(), want1.cpu().numpy()) < OP_TOL
    assert rel(got2.cpu().numpy(), want2.cpu().numpy()) < OP_TOL
    assert torch.equal(got1, want1) and torch.equal(got2, want2)            # same kernel, same arithmetic: same bits
    # and against the oracle's own FFT on sampled frames, so that this file stands on its own
    for i in (0, 17, K - 1):
        assert rel(got1[i].cpu().numpy(), oracle.fft2(f1[i].cpu().numpy(), -1)) < OP_TOL
        assert rel(got2[i].cpu().numpy(), oracle.fft2(f2[i].cpu().numpy(), +1)) < OP_TOL
    # a third call with fewer frames than clusters, repeating call 1's data: same result again
    sharp.fft2_noalloc(f1[:3].contiguous(), out[:3], -1)
    assert torch.equal(out[:3], want1[:3])
    rec.close()


def test_noalloc_fft2_rejects_what_it_cannot_do():
    import torch
    f = torch.zeros((2, M, M), dtype=torch.complex64, device="cuda")
    out = torch.empty_like(f)
    lib = sharp.load_library()
    import ctypes as C
    st = C.c_void_p(torch.cuda.current_stream().cuda_stream)
    p = lambda t: C.c_void_p(t.data_ptr())
    # beyond the static scratch's stated maximum: refused before anything is launched
    assert lib.sharp_fft2_noalloc(p(f), p(out), M, sharp.NOALLOC_MAX_FRAMES + 1, -1, st) == sharp.SHARP_EINVAL
    assert b"4096" in lib.sharp_last_error(None)
    assert lib.sharp_fft2_noalloc(p(f), p(out), 128, 2, -1, st) == sharp.SHARP_EINVAL          # m = 256 only
    assert lib.sharp_fft2_noalloc(p(f), p(f), M, 2, -1, st) == sharp.SHARP_EINVAL              # out of place
    assert lib.sharp_fft2_noalloc(p(f), p(out), M, 2, 0, st) == sharp.SHARP_EINVAL             # sign
    assert lib.sharp_fft2_noalloc(p(f), None, M, 2, -1, st) == sharp.SHARP_EINVAL
    assert lib.sharp_fft2_noalloc(p(f), p(out), M, 2, -1, st) == sharp.SHARP_OK                # and it still works
    torch.cuda.synchronize()
    assert float(out.abs().max()) == 0.0
