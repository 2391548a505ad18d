"""Pins of the F-engine oracle (oracle/fengine.py; Eq. 1, FFT length 256 PAPER.md:176).  CPU only."""
import numpy as np
import pytest

from oracle import fengine as fo

L = fo.FFT_LEN


def _rand(rng, M, A):
    return rng.integers(-128, 128, size=(M, A * L), dtype=np.int8)


def test_matches_library_rfft():
    rng = np.random.default_rng(1)
    s = _rand(rng, 5, 3)
    S = fo.fengine(s)
    ref = np.fft.rfft(s.reshape(5, 3, L).astype(np.float64), axis=-1)[..., :L // 2]     # [m][a][k]
    assert S.shape == (3, L // 2, 5)
    assert np.allclose(S, ref.transpose(1, 2, 0), rtol=0, atol=1e-8)


def test_impulse_constant_and_shift():
    s = np.zeros((3, L), np.int8)
    s[0, 0] = 7                    # impulse at n = 0: flat spectrum 7
    s[1, :] = -3                   # constant: only the DC channel, N * value
    s[2, 5] = 9                    # impulse at n = 5: 9 exp(-j 2 pi 5 k / N)
    S = fo.fengine(s)[0]
    k = np.arange(L // 2)
    assert np.allclose(S[:, 0], 7)
    assert np.allclose(S[0, 1], -3 * L) and np.allclose(S[1:, 1], 0, atol=1e-9)
    assert np.allclose(S[:, 2], 9 * np.exp(-2j * np.pi * 5 * k / L), atol=1e-10)


def test_real_tone_closed_form():
    """s[n] = round(100 cos(2 pi k0 n / N)) is not exactly a tone; use the exact definition on an exactly
    representable two-level signal instead: s[n] = (-1)^n * 64 has S[k] = 0 for every kept channel (it lives in the
    dropped Nyquist bin), and s[n] = 64 for n even, 0 for n odd gives S[0] = 64 N / 2 and zero elsewhere."""
    n = np.arange(L)
    s = np.stack([np.where(n % 2 == 0, 64, -64), np.where(n % 2 == 0, 64, 0)]).astype(np.int8)
    S = fo.fengine(s)[0]
    assert np.allclose(S[:, 0], 0, atol=1e-9)
    assert np.allclose(S[0, 1], 64 * L / 2) and np.allclose(S[1:, 1], 0, atol=1e-9)


def test_quarter_rate_tone_sign_of_the_exponent():
    """s[n] = 100 cos(pi n / 2) + 50 sin(pi n / 2) takes the exact values (100, 50, -100, -50): the whole signal sits in
    channel k = N/4 with S = (N/2) (100 - 50 j): the MINUS sign of Eq. 1's exponent is what makes the sine part -j."""
    n = np.arange(L)
    s = np.array([100, 50, -100, -50], np.int8)[n % 4][None, :]
    S = fo.fengine(np.ascontiguousarray(s))[0, :, 0]
    want = np.zeros(L // 2, complex)
    want[L // 4] = (L / 2) * (100 - 50j)
    assert np.allclose(S, want, atol=1e-9)


def test_linearity_parseval_and_block_independence():
    rng = np.random.default_rng(2)
    a, b = _rand(rng, 2, 4) // 2, _rand(rng, 2, 4) // 2
    assert np.allclose(fo.fengine((a + b).astype(np.int8)), fo.fengine(a.astype(np.int8)) + fo.fengine(b.astype(np.int8)), atol=1e-8)
    s = _rand(rng, 1, 4)
    S = fo.fengine(s)
    # Parseval on the full (Hermitian) spectrum: sum|s|^2 = (|S0|^2 + |S_Nyq|^2 + 2 sum_{0<k<N/2} |S_k|^2) / N
    blk = s.reshape(4, L).astype(np.float64)
    nyq = (blk * (-1.0) ** np.arange(L)).sum(axis=1)
    lhs = (blk ** 2).sum(axis=1)
    rhs = (np.abs(S[:, 0, 0]) ** 2 + nyq ** 2 + 2 * (np.abs(S[:, 1:, 0]) ** 2).sum(axis=1)) / L
    assert np.allclose(lhs, rhs, rtol=1e-12)
    # block a depends only on samples [a N, (a+1) N)
    s2 = s.copy(); s2[0, 2 * L:3 * L] = 0
    S2 = fo.fengine(s2)
    assert np.allclose(S2[[0, 1, 3]], S[[0, 1, 3]]) and np.allclose(S2[2], 0)


def test_layout_and_fp16_rounding():
    rng = np.random.default_rng(3)
    s = _rand(rng, 6, 2)
    S = fo.fengine(s)
    x = fo.to_xengine_input(S)
    assert x.shape == (2, L // 2, 6, 2) and x.dtype == np.float16
    assert np.abs(S).max() <= 128 * L < 65504                 # every spectrum value is finite in fp16 (F-engine reading)
    assert (np.abs(x[..., 0].astype(np.float64) - S.real) <= 0.5 * np.spacing(np.abs(x[..., 0]).astype(np.float16)).astype(np.float64) + 1e-12).all()


def test_to_xengine_input_rounds_both_components_to_nearest_even():
    """Hand-written half-way cases (binary16 has 11 significant bits: spacing 2 in [2048, 4096), 4 in [4096, 8192)):
    2049 -> 2048 and 2051 -> 2052 (ties to even), 2050 exact, 4098 -> 4096, 4102 -> 4104, -2049 -> -2048; the real and the
    imaginary part are rounded independently and land in [..., 0] and [..., 1]."""
    S = np.array([[[2049 + 2051j, 2051 - 2049j, 2050 + 4098j, -2049 + 4102j, 0.1 - 65504j, 1e-9 + 3j]]])        # [1, 1, 6]
    x = fo.to_xengine_input(S)
    assert x.shape == (1, 1, 6, 2) and x.dtype == np.float16
    want = [[2048, 2052], [2052, -2048], [2050, 4096], [-2048, 4104], [float(np.float16(0.1)), -65504], [0.0, 3]]
    got = x[0, 0].astype(np.float64)
    assert got[:5].tolist() == want[:5]
    assert got[5, 1] == 3 and abs(got[5, 0] - 1e-9) < 6e-8 and got[5, 0] in (0.0, float(np.float16(1e-9)))     # below the subnormal step
    assert float(np.float16(0.1)) == 0.0999755859375            # 0.1 -> nearest binary16, written out


def test_rejects_bad_input():
    with pytest.raises(ValueError):
        fo.fengine(np.zeros((2, 100), np.int8))
    with pytest.raises(ValueError):
        fo.fengine(np.zeros((2, L), np.int16))


def test_quantise_ci8_rounding_clipping_and_tie_distance():
    """clip(rint(S * scale), +-127): ties go to even (numpy rint and the kernel's cvt.rni agree on that), -128 is never
    produced, and the reported tie distance is 0 exactly at k + 0.5."""
    S = np.array([[[0.5 + 1.5j, 2.5 - 0.5j, 2.49 + 2.51j, 1000 - 1000j, -127.4 + 127.6j, 3.0 - 3.0j]]])   # [1, 1, 6]
    codes, tie = fo.quantise_ci8(S, 1.0)
    assert codes.dtype == np.int8 and codes.shape == (1, 1, 6, 2)
    assert codes[0, 0].tolist() == [[0, 2], [2, 0], [2, 3], [127, -127], [-127, 127], [3, -3]]
    assert tie[0, 0, 0, 0] == 0 and tie[0, 0, 1, 0] == 0 and abs(tie[0, 0, 5, 0] - 0.5) < 1e-12
    codes2, _ = fo.quantise_ci8(S, 0.5)
    assert codes2[0, 0, 3].tolist() == [127, -127] and codes2[0, 0, 5].tolist() == [2, -2]        # 1.5 -> 2, -1.5 -> -2
