"""corr_xengine_static -- the X-engine entry point that allocates nothing (include/corr.h).

Why the library has it: some of its users cannot call cudaMalloc when they need a correlation.  A real-time capture
process hands all GPU memory to its ring buffers at start-up and must not stall the device later (cudaMalloc / cudaFree
synchronise it); a plug-in may live in a host application that forbids driver allocations after initialisation.  For them
the pair kernel's scratch (tile table + tile-feed counter) sits in a fixed 16.5 KB array inside libcorr.so instead of in
memory that corr_create allocates.

What is checked here: on two calls in a row -- which share that array, the second finding the first one's leftovers in
it -- the result equals the existing handle path (corr_create + corr_xengine on the same kernel): bit for bit on the int8
path, within the fp16 tolerance of the parity tests (2e-5 normalised; in practice also bit for bit) on the fp16 path.
The geometries differ between the two calls so that a stale tile table or a counter that was not cleared would show.
Problems larger than the array are refused with a message that names the limit.

This file sorts last on purpose (pytest -x stops at the first failure: a failure here must not hide other tests) and
depends on nothing the other tests leave behind: it passes alone in a fresh process and after the whole suite.
"""
import ctypes

import numpy as np
import pytest
import torch

from paper_1305_5639_b200 import inputs

FP16_TOL = 2e-5          # as tests/test_parity_gpu.py


@pytest.fixture(scope="module")
def corr():
    from paper_1305_5639_b200 import binding
    binding.lib()
    return binding


def _handle_path(corr, x, dtype, prev=None):
    """The existing path on the same kernel: corr_create + corr_set_kernel(PAIR) + corr_xengine."""
    T, C, N, P, _ = x.shape
    with corr.Correlator(N, P, C, T, dtype) as h:
        h.set_kernel("pair")
        out = h.xengine(x, prev.clone() if prev is not None else None, accumulate=prev is not None)
        torch.cuda.synchronize()
    return out


def _normalised_error(got, want, N, P):
    """max |dV_ij| / sqrt(V_ii^pp V_jj^qq), autocorrelations taken from `want`."""
    got, want = got.double().cpu().numpy(), want.double().cpu().numpy()
    i_of_b = np.concatenate([np.full(i + 1, i) for i in range(N)])
    j_of_b = np.concatenate([np.arange(i + 1) for i in range(N)])
    auto_b = np.array([i * (i + 1) // 2 + i for i in range(N)])
    auto = np.stack([want[:, auto_b, p, p, 0] for p in range(P)], axis=-1)
    d = got - want
    err = np.sqrt(d[..., 0] ** 2 + d[..., 1] ** 2)
    return float((err / np.sqrt(auto[:, i_of_b, :, None] * auto[:, j_of_b, None, :])).max())


@pytest.mark.gpu
def test_static_entry_point_matches_handle_path_int8(corr):
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (there is no CPU fallback)")
    # call 1: N = 200, two pols -> 800 components = 4 row blocks (10 tiles per channel), ragged last block, many tiles
    # per cluster; call 2, straight after it on the same stream: N = 72 -> 2 row blocks (3 tiles per channel), so the array
    # still holds call 1's longer table and its spent counter when call 2 prepares it
    x1 = inputs.gauss_ci8(300, 40, 200, 2, 30.0, seed=11).cuda()
    x2 = inputs.gauss_ci8(520, 9, 72, 2, 30.0, seed=12).cuda()
    got1 = corr.xengine_static(x1)
    got2 = corr.xengine_static(x2)
    torch.cuda.synchronize()
    want1, want2 = _handle_path(corr, x1, "ci8"), _handle_path(corr, x2, "ci8")
    assert torch.equal(got1, want1), "call 1 differs in %d words" % int((got1 != want1).sum())
    assert torch.equal(got2, want2), "call 2 differs in %d words" % int((got2 != want2).sum())
    # and integrating a further block into call 2's result (accumulate), again back to back with a different geometry first
    x3 = inputs.gauss_ci8(520, 9, 72, 2, 30.0, seed=13).cuda()
    corr.xengine_static(x1, got1)                       # rewrites the array for N = 200
    corr.xengine_static(x3, got2, accumulate=True)      # ... and this call must put N = 72's table back
    torch.cuda.synchronize()
    assert torch.equal(got1, want1)
    assert torch.equal(got2, _handle_path(corr, x3, "ci8", prev=want2))


@pytest.mark.gpu
def test_static_entry_point_matches_handle_path_fp16(corr):
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (there is no CPU fallback)")
    N1, N2, P = 96, 40, 2
    x1 = inputs.corr_phase_cf16(1100, 6, N1, P, seed=21).cuda()      # more than one 1024-sample accumulation pass
    x2 = inputs.corr_phase_cf16(200, 5, N2, P, seed=22).cuda()
    got1 = corr.xengine_static(x1)
    got2 = corr.xengine_static(x2)
    torch.cuda.synchronize()
    want1, want2 = _handle_path(corr, x1, "cf16"), _handle_path(corr, x2, "cf16")
    assert _normalised_error(got1, want1, N1, P) <= FP16_TOL
    assert _normalised_error(got2, want2, N2, P) <= FP16_TOL


def test_static_entry_point_refuses_what_the_array_cannot_hold(corr):
    """Argument checks come before any CUDA call, so this runs without a GPU (the pointers are never touched)."""
    L = corr.lib()
    assert L.corr_static_scratch_bytes() == 4 * (64 + 2 * 2080)
    fake = ctypes.c_void_p(1 << 20)          # 16-byte aligned, never dereferenced
    rc = L.corr_xengine_static(corr.STATIC_MAX_STREAMS // 2 + 1, 2, 1, 64, corr.CORR_CI8, fake, fake, 0, None)
    assert rc == corr.CORR_EINVAL
    msg = L.corr_last_error(None).decode()
    assert "CORR_STATIC_MAX_STREAMS = 8192" in msg and "corr_create" in msg
    # a row TMA cannot address is refused too (no CUDA-core fallback on this path), as is an int8 overflow
    assert L.corr_xengine_static(9, 1, 1, 64, corr.CORR_CI8, fake, fake, 0, None) == corr.CORR_EUNSUPPORTED
    assert L.corr_xengine_static(16, 2, 1, 65536, corr.CORR_CI8, fake, fake, 0, None) == corr.CORR_EOVERFLOW
    assert L.corr_xengine_static(16, 2, 1, 64, corr.CORR_CI8, None, fake, 0, None) == corr.CORR_EINVAL
