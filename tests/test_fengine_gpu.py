"""GPU parity of corr_fengine (Eq. 1, N = 256) against the fp64 DFT-definition oracle, and the F -> X chain.

Tolerance: the kernel computes in fp32 and rounds once to fp16, the oracle is exact to fp64:
    |d component| <= 0.5 ulp_fp16(|exact component|) + 2e-6 * sum_n |s[n]|
(the first term is the one rounding to the fp16 output format, the second bounds the fp32 round-off of an 8-stage
256-point transform: log2(256) * 2^-23 * sum|s| = 9.5e-7 sum|s|, doubled).
"""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def corr():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (there is no CPU fallback)")
    from paper_1305_5639_b200 import binding
    binding.lib()
    return binding


def check(corr, s, simt=False):
    from oracle import fengine as fo
    got = corr.fengine(torch.from_numpy(s).cuda(), simt=simt).cpu().numpy().astype(np.float64)       # [A, 128, M, 2]
    want = fo.fengine(s)
    A, K, M = want.shape
    assert got.shape == (A, K, M, 2)
    l1 = np.abs(s.reshape(M, A, 256).astype(np.float64)).sum(axis=2).T[:, None, :]         # [A, 1, M]
    for part, w in ((0, want.real), (1, want.imag)):
        ulp = np.spacing(np.abs(w).astype(np.float16)).astype(np.float64)
        tol = 0.5 * ulp + 2e-6 * l1
        bad = np.argwhere(np.abs(got[..., part] - w) > tol)
        assert bad.size == 0, "part %d first mismatches (a,k,m): %s" % (part, bad[:6].tolist())


@pytest.mark.parametrize("M,A", [(1, 1), (2, 3), (7, 2), (24, 3), (32, 4), (33, 5), (64, 16), (100, 9), (512, 8)])
def test_fengine_random_full_range(corr, M, A):
    rng = np.random.default_rng(9000 + M)
    s = rng.integers(-128, 128, size=(M, A * 256), dtype=np.int8)
    # tensor cores: rows 16-byte aligned (M % 8 == 0) and a ragged last half tile that at most doubles the work
    assert corr.fengine_uses_tensor_cores(M) == (M % 8 == 0 and -(-M // 64) * 64 <= 2 * M)
    check(corr, s)
    check(corr, s, simt=True)                            # the CUDA-core kernel on the same input


@pytest.mark.parametrize("M,A", [(64, 1), (64, 149), (128, 33), (192, 7), (320, 2), (512, 300), (1024, 37),
                                 (32, 5), (40, 7), (72, 149), (96, 33), (200, 3), (456, 21)])
def test_fengine_tensor_core_path(corr, M, A):
    """The tcgen05 kernel (whole half tiles of 64 streams, and stream counts with a RAGGED last half tile -- 72 and 96 used to
    fall back to the CUDA-core kernel): more tiles than SMs, a single tile, odd tile counts;
    full-range int8 including -128; the same bound as the CUDA-core kernel, and the two kernels agree to one fp16 ulp
    plus both fp32 round-off allowances."""
    rng = np.random.default_rng(9100 + M + A)
    s = rng.integers(-128, 128, size=(M, A * 256), dtype=np.int8)
    assert corr.fengine_uses_tensor_cores(M)
    check(corr, s)
    sd = torch.from_numpy(s).cuda()
    tc, cc = corr.fengine(sd).float(), corr.fengine(sd, simt=True).float()
    big = torch.maximum(tc.abs(), cc.abs()).cpu().numpy()
    ulp = np.spacing(big.astype(np.float16)).astype(np.float64)
    l1 = np.abs(s.reshape(M, A, 256).astype(np.float64)).sum(axis=2).T[:, None, :, None]          # [A, 1, M, 1]
    assert ((tc - cc).abs().cpu().numpy() <= ulp + 4e-6 * l1).all()


def test_fengine_tensor_core_exact_cases(corr):
    """64 streams of hand-checkable inputs through the tcgen05 kernel: impulses at n = 0, 1, 128 (the sample that bypasses
    the folded sums), 200; DC; extreme DC; the Nyquist tone (dropped bin); a full-scale tone on a bin centre."""
    n = np.arange(512)
    s = np.zeros((64, 512), np.int8)
    s[0, 0] = 7; s[0, 256 + 5] = 9
    s[1, :] = -3
    s[2, :] = np.array([100, 50, -100, -50])[n % 4]
    s[3, :] = 127; s[4, :] = -128
    s[5, :] = np.where(n % 2 == 0, 127, -128)
    s[6, 128] = 11; s[6, 256 + 1] = -5
    s[7, :] = np.rint(127 * np.cos(2 * np.pi * 37 * n / 256)).astype(np.int8)
    s[8:] = np.random.default_rng(3).integers(-128, 128, size=(56, 512), dtype=np.int8)
    assert corr.fengine_uses_tensor_cores(64)
    got = corr.fengine(torch.from_numpy(s).cuda()).cpu().numpy().astype(np.float64)
    assert (got[0, :, 0, 0] == 7).all() and (got[0, :, 0, 1] == 0).all()
    assert got[0, 0, 1, 0] == -768 and np.abs(got[:, 1:, 1]).max() <= 1e-3
    assert got[1, 64, 2, 0] == 12800 and got[1, 64, 2, 1] == -6400
    assert got[0, 0, 3, 0] == 127 * 256 and got[0, 0, 4, 0] == -128 * 256
    assert got[0, 0, 5, 0] == -128 and np.abs(got[:, 1:, 5]).max() <= 0.05
    assert (got[0, :, 6, 0] == 11 * np.where(np.arange(128) % 2 == 0, 1, -1)).all() and (got[0, :, 6, 1] == 0).all()
    check(corr, s)


def test_fengine_exact_cases(corr):
    n = np.arange(512)
    s = np.zeros((6, 512), np.int8)
    s[0, 0] = 7; s[0, 256 + 5] = 9                       # impulses
    s[1, :] = -3                                         # DC
    s[2, :] = np.array([100, 50, -100, -50])[n % 4]      # quarter-rate tone: channel 64 = 128 (100 - 50 j)
    s[3, :] = 127; s[4, :] = -128                        # extreme DC: 32512 and -32768 are exact in fp16
    s[5, :] = np.where(n % 2 == 0, 127, -128)            # lives in the dropped Nyquist bin (+ DC -128)
    got = corr.fengine(torch.from_numpy(s).cuda()).cpu().numpy().astype(np.float64)
    assert (got[0, :, 0, 0] == 7).all() and (got[0, :, 0, 1] == 0).all()
    assert got[0, 0, 1, 0] == -768 and np.abs(got[:, 1:, 1]).max() <= 1e-3
    assert got[1, 64, 2, 0] == 12800 and got[1, 64, 2, 1] == -6400
    assert got[0, 0, 3, 0] == 127 * 256 and got[0, 0, 4, 0] == -128 * 256
    assert got[0, 0, 5, 0] == -128 and np.abs(got[:, 1:, 5]).max() <= 0.05
    check(corr, s)


def test_fengine_then_xengine_chain(corr):
    """F-engine output is consumed in place by the fp16 X-engine (no corner turn): the visibilities equal the X-engine
    oracle applied to the F-engine's own fp16 output, within the X-engine tolerance."""
    import oracle
    N, P, A = 24, 2, 192
    rng = np.random.default_rng(77)
    s = np.clip(np.rint(rng.normal(0, 20, size=(N * P, A * 256))), -127, 127).astype(np.int8)
    x = corr.fengine(torch.from_numpy(s).cuda())                             # [A, 128, N*P, 2] fp16
    x5 = x.view(A, 128, N, P, 2)
    with corr.Correlator(N, P, 128, A, "cf16") as h:
        got = h.xengine(x5).cpu().numpy().astype(np.float64)
    want = oracle.xengine(x5.cpu().numpy())
    auto_b = np.array([i * (i + 1) // 2 + i for i in range(N)])
    i_of_b = np.concatenate([np.full(i + 1, i) for i in range(N)]); j_of_b = np.concatenate([np.arange(i + 1) for i in range(N)])
    auto = np.stack([want[:, auto_b, p, p, 0] for p in range(P)], axis=-1)
    d = got - want
    err = np.sqrt(d[..., 0] ** 2 + d[..., 1] ** 2) / np.sqrt(auto[:, i_of_b, :, None] * auto[:, j_of_b, None, :])
    assert err[1:].max() <= 2e-5            # channel 0 (DC) of zero-mean noise has tiny autocorrelations; skip its ratio


def test_fengine_argument_errors(corr):
    L = corr.lib()
    s = torch.zeros((4, 512), dtype=torch.int8, device="cuda")
    out = torch.empty((2, 128, 4, 2), dtype=torch.float16, device="cuda")
    assert L.corr_fengine(None, out.data_ptr(), 4, 2, None) == corr.CORR_EINVAL
    assert L.corr_fengine(s.data_ptr(), out.data_ptr(), 0, 2, None) == corr.CORR_EINVAL
    assert L.corr_fengine(s.data_ptr() + 1, out.data_ptr(), 4, 2, None) == corr.CORR_EINVAL
    assert b"corr_fengine" in L.corr_last_error(None)
    with pytest.raises(ValueError):
        corr.fengine(torch.zeros((4, 500), dtype=torch.int8, device="cuda"))


# ---- requantised int8 output (corr_fengine_ci8): the code is decided by rint of an fp32 product on the GPU and of an
# fp64 product in the oracle, so the two must agree EXACTLY except where the scaled value lies within the fp32 round-off
# bound of a rounding tie, and there they may differ by one code (quantised decisions) ----
# (stream counts that are a multiple of 8, at least 32, run on the tensor-core kernel, the others on the CUDA-core kernel)
@pytest.mark.parametrize("M,A,scale", [(2, 3, 1.0 / 64), (33, 4, 1.0 / 40), (64, 8, 0.05), (100, 5, 1.0 / 300),
                                       (128, 33, 1.0 / 40), (192, 7, 1.0 / 25), (512, 40, 1.0 / 64),
                                       (40, 9, 1.0 / 40), (72, 150, 1.0 / 30), (96, 33, 0.05), (200, 7, 1.0 / 64)])
def test_fengine_ci8_codes(corr, M, A, scale):
    from oracle import fengine as fo
    rng = np.random.default_rng(9100 + M)
    s = np.clip(np.rint(rng.normal(0, 25, size=(M, A * 256))), -127, 127).astype(np.int8)
    got = corr.fengine(torch.from_numpy(s).cuda(), scale=scale).cpu().numpy()
    S = fo.fengine(s)
    want, tie = fo.quantise_ci8(S, scale)
    assert got.dtype == np.int8 and got.shape == want.shape
    l1 = np.abs(s.reshape(M, A, 256).astype(np.float64)).sum(axis=2).T[:, None, :, None]      # [A, 1, M, 1]
    near_tie = tie <= (2e-6 * l1 + 1e-6 * np.abs(np.stack([S.real, S.imag], -1))) * scale + 1e-7
    diff = got.astype(np.int16) - want.astype(np.int16)
    assert (diff[~near_tie] == 0).all()
    assert (np.abs(diff[near_tie]) <= 1).all()
    assert near_tie.mean() < 5e-3                      # the tie band is tiny: the test is essentially exact
    assert got.min() >= -127


def test_fengine_ci8_then_int8_xengine_chain(corr):
    """The whole int8 FX pair on the GPU: samples -> corr_fengine_ci8 -> corr_xengine (CORR_CI8); the X-engine stage is
    bit-exact against the oracle on the F-engine's own codes."""
    import oracle
    N, P, A = 40, 2, 128
    rng = np.random.default_rng(78)
    s = np.clip(np.rint(rng.normal(0, 20, size=(N * P, A * 256))), -127, 127).astype(np.int8)
    x = corr.fengine(torch.from_numpy(s).cuda(), scale=1.0 / 20)                 # sigma ~ 16 codes per component
    assert 8 < x.float().std().item() < 24
    x5 = x.view(A, 128, N, P, 2)
    with corr.Correlator(N, P, 128, A, "ci8") as h:
        got = h.xengine(x5).cpu().numpy().astype(np.int64)
    assert (got == oracle.xengine(x5.cpu().numpy())).all()


def test_fengine_ci8_argument_errors(corr):
    L = corr.lib()
    s = torch.zeros((4, 512), dtype=torch.int8, device="cuda")
    out = torch.empty((2, 128, 4, 2), dtype=torch.int8, device="cuda")
    assert L.corr_fengine_ci8(s.data_ptr(), out.data_ptr(), 4, 2, 0.0, None) == corr.CORR_EINVAL
    assert L.corr_fengine_ci8(s.data_ptr(), None, 4, 2, 1.0, None) == corr.CORR_EINVAL
    assert L.corr_fengine_ci8(s.data_ptr(), out.data_ptr() + 1, 4, 2, 1.0, None) == corr.CORR_EINVAL
