"""Pins for the CPU oracle (oracle/xengine_oracle.c) against what the paper and mathematics fix.

The paper prints no numerical X-engine output, so every pin is Eq. 2 evaluated by
a route that is structurally different from the oracle's loops: a hand-worked example, numpy
complex128 einsum / matmul (ZGEMM), closed forms, and invariants.  Each pin is chosen so that a
plausible slip in the oracle (conjugating the wrong factor, a sign in Im, swapped polarisation
axes, a wrong baseline index, a dropped term) fails at least one of them.
"""
import os

import numpy as np
import pytest

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def to_complex(x):
    x = np.asarray(x)
    return x[..., 0].astype(np.float64) + 1j * x[..., 1].astype(np.float64)


def full_matrix_numpy(x):
    """H[c, m, n] = sum_t conj(x[t,c,m]) x[t,c,n] via complex128 einsum, m = s*P+p."""
    T, C, N, P, _ = x.shape
    z = to_complex(x).reshape(T, C, N * P)
    return np.einsum("tcm,tcn->cmn", np.conj(z), z)


def pack(H, N, P):
    """[C, M, M] complex -> [C, B, P, P] complex with b = i(i+1)/2+j, written out independently."""
    C = H.shape[0]
    V = np.zeros((C, N * (N + 1) // 2, P, P), dtype=np.complex128)
    b = 0
    for i in range(N):
        for j in range(i + 1):
            V[:, b] = H[:, i * P:(i + 1) * P, j * P:(j + 1) * P]
            b += 1
    return V


def rand_ci8(rng, T, C, N, P, lo=-127, hi=127):
    return rng.integers(lo, hi + 1, size=(T, C, N, P, 2), dtype=np.int8)


# ---- pin 0: hand-worked example -------------------------------------------------------------
def test_hand_worked_example(oracle):
    sect, inp, exp = None, [], []
    for line in open(os.path.join(GOLD, "eq2_hand_example.txt")):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        if line in ("input", "expected"):
            sect = line
            continue
        (inp if sect == "input" else exp).append([int(v) for v in line.split()])
    x = np.zeros((2, 1, 2, 1, 2), dtype=np.int8)
    for t, s, re, im in inp:
        x[t, 0, s, 0] = (re, im)
    V = oracle.xengine(x)
    assert V.shape == (1, 3, 1, 1, 2) and V.dtype == np.int64
    for b, i, j, re, im in exp:
        assert oracle.baseline_index(i, j) == b
        assert tuple(V[0, b, 0, 0]) == (re, im)
        assert oracle.visibility(x, 0, i, 0, j, 0) == (re, im)


# ---- pin 1: brute force on tiny inputs, two independent routes ------------------------------
@pytest.mark.parametrize("N,P,C,T", [(1, 1, 1, 1), (2, 2, 1, 3), (3, 1, 2, 8), (4, 2, 2, 5)])
def test_tiny_bruteforce(oracle, N, P, C, T):
    rng = np.random.default_rng(100 + N * 10 + P)
    x = rand_ci8(rng, T, C, N, P, -9, 9)
    V = oracle.xengine(x)
    # route A: numpy einsum
    ref = pack(full_matrix_numpy(x), N, P)
    assert np.array_equal(V[..., 0], np.rint(ref.real).astype(np.int64))
    assert np.array_equal(V[..., 1], np.rint(ref.imag).astype(np.int64))
    # route B: pure-Python complex arithmetic, one term at a time
    for c in range(C):
        for i in range(N):
            for j in range(i + 1):
                for p in range(P):
                    for q in range(P):
                        acc = 0j
                        for t in range(T):
                            a = complex(int(x[t, c, i, p, 0]), int(x[t, c, i, p, 1]))
                            b = complex(int(x[t, c, j, q, 0]), int(x[t, c, j, q, 1]))
                            acc += a.conjugate() * b
                        got = V[c, i * (i + 1) // 2 + j, p, q]
                        assert (got[0], got[1]) == (acc.real, acc.imag)


# ---- pin 2: reduction to a library ZGEMM ----------------------------------------------------
def test_reduces_to_zgemm(oracle):
    rng = np.random.default_rng(2)
    T, C, N, P = 97, 3, 11, 2
    x = rand_ci8(rng, T, C, N, P)
    V = oracle.xengine(x)
    z = to_complex(x).reshape(T, C, N * P)
    for c in range(C):
        Xc = z[:, c, :]
        H = Xc.conj().T @ Xc                       # ZGEMM, exact: all sums < 2^53
        ref = pack(H[None], N, P)[0]
        assert np.array_equal(V[c, ..., 0], np.rint(ref.real).astype(np.int64))
        assert np.array_equal(V[c, ..., 1], np.rint(ref.imag).astype(np.int64))


def test_cf16_reduces_to_zgemm(oracle):
    rng = np.random.default_rng(22)
    T, C, N, P = 64, 2, 6, 2
    x = rng.standard_normal((T, C, N, P, 2)).astype(np.float16)
    V = oracle.xengine(x)
    assert V.dtype == np.float64
    ref = pack(full_matrix_numpy(x), N, P)
    scale = np.abs(ref).max()
    assert np.max(np.abs(V[..., 0] + 1j * V[..., 1] - ref)) <= 1e-12 * scale
    # the single-visibility routine on fp16 input (xo_pair_cf16) against the same ZGEMM entries, every (c, i, p, j, q)
    for c in range(C):
        for i in range(N):
            for j in range(i + 1):
                for p in range(P):
                    for q in range(P):
                        re, im = oracle.visibility(x, c, i, p, j, q)
                        assert abs(complex(re, im) - ref[c, oracle.baseline_index(i, j), p, q]) <= 1e-12 * scale


def test_half_conversion_all_patterns(oracle):
    bits = np.arange(65536, dtype=np.uint16)
    lib = bits.view(np.float16).astype(np.float64)           # numpy's converter, independent
    for b in range(65536):                                   # every binary16 pattern, NaNs and subnormals included
        got = oracle.half_to_double(b)
        assert (np.isnan(got) and np.isnan(lib[b])) or got == lib[b]
    assert np.signbit(oracle.half_to_double(0x8000))


# ---- pin 3: Hermitian symmetry --------------------------------------------------------------
def test_hermitian_symmetry(oracle):
    rng = np.random.default_rng(3)
    T, C, N, P = 33, 2, 5, 2
    x = rand_ci8(rng, T, C, N, P)
    V = oracle.xengine(x)
    for c in range(C):
        for i in range(N):
            for j in range(N):
                for p in range(P):
                    for q in range(P):
                        vij = oracle.visibility(x, c, i, p, j, q)
                        vji = oracle.visibility(x, c, j, q, i, p)
                        assert vji == (vij[0], -vij[1])
                        if j <= i:
                            assert tuple(V[c, oracle.baseline_index(i, j), p, q]) == vij
            b = oracle.baseline_index(i, i)     # packed: V_ii^{XY} = conj(V_ii^{YX})
            assert V[c, b, 0, 1, 0] == V[c, b, 1, 0, 0] and V[c, b, 0, 1, 1] == -V[c, b, 1, 0, 1]


# ---- pin 4: autocorrelations are real and non-negative --------------------------------------
def test_autocorrelations(oracle):
    rng = np.random.default_rng(4)
    T, C, N, P = 50, 2, 6, 2
    x = rand_ci8(rng, T, C, N, P)
    V = oracle.xengine(x)
    power = (x.astype(np.int64) ** 2).sum(axis=(0, 4))       # [C, N, P]
    for i in range(N):
        b = oracle.baseline_index(i, i)
        for p in range(P):
            assert np.all(V[:, b, p, p, 1] == 0)
            assert np.array_equal(V[:, b, p, p, 0], power[:, i, p])
            assert np.all(V[:, b, p, p, 0] >= 0)


# ---- pin 5: constant input closed form, asymmetric constants --------------------------------
def test_constant_closed_form(oracle):
    T, C, N, P = 37, 2, 3, 2
    a = np.array([[3 + 4j, -2 + 7j], [5 - 1j, -6 - 2j], [0 + 9j, 8 + 0j]])   # [N, P]
    x = np.zeros((T, C, N, P, 2), dtype=np.int8)
    x[..., 0] = a.real
    x[..., 1] = a.imag
    V = oracle.xengine(x)
    for i in range(N):
        for j in range(i + 1):
            for p in range(P):
                for q in range(P):
                    v = T * np.conj(a[i, p]) * a[j, q]       # = T * a_j * conj(b_i): north_star's form
                    got = V[:, oracle.baseline_index(i, j), p, q]
                    assert np.all(got[:, 0] == v.real) and np.all(got[:, 1] == v.imag)
    # the sign of Im is pinned by an explicit number: conj(3+4j)(-2+7j) = 22+29j
    assert tuple(V[0, oracle.baseline_index(0, 0), 0, 1]) == (22 * T, 29 * T)


# ---- pin 6: identical streams ---------------------------------------------------------------
def test_identical_streams(oracle):
    rng = np.random.default_rng(6)
    T, C, N, P = 40, 2, 4, 1
    one = rand_ci8(rng, T, C, 1, P)
    x = np.repeat(one, N, axis=2)
    V = oracle.xengine(x)
    for b in range(V.shape[1]):
        assert np.array_equal(V[:, b], V[:, 0])
    assert np.all(V[..., 1] == 0)


# ---- pin 7: single tone with a per-station delay: analytic phase ----------------------------
def test_delayed_tone_exact_quarter_turns(oracle):
    # phases that are multiples of pi/2 are exact in fp16 and int8: V_ij = T * e^{+j 2 pi f (tau_i - tau_j)}
    T, C, N, P = 16, 4, 4, 1
    turns = np.array([[(c * s) % 4 for s in range(N)] for c in range(C)])     # f_c * tau_s in quarter turns
    ph = np.exp(-2j * np.pi * turns / 4.0)                                    # x_s = e^{-j 2 pi f tau_s}
    x = np.zeros((T, C, N, P, 2), dtype=np.float16)
    x[..., 0, 0] = np.rint(ph.real)
    x[..., 0, 1] = np.rint(ph.imag)
    V = oracle.xengine(x)
    Vi = oracle.xengine((x * 100).astype(np.int8))
    for c in range(C):
        for i in range(N):
            for j in range(i + 1):
                want = T * np.exp(+2j * np.pi * (turns[c, i] - turns[c, j]) / 4.0)
                got = V[c, oracle.baseline_index(i, j), 0, 0]
                assert abs(complex(got[0], got[1]) - want) < 1e-12
                goti = Vi[c, oracle.baseline_index(i, j), 0, 0]
                assert abs(complex(goti[0], goti[1]) - 1e4 * want) < 1e-9
                # xo_pair_cf16 / xo_pair_ci8 straight from the ungathered input: the same closed form (sign of Im pinned)
                assert abs(complex(*oracle.visibility(x, c, i, 0, j, 0)) - want) < 1e-12
                assert abs(complex(*oracle.visibility((x * 100).astype(np.int8), c, i, 0, j, 0)) - 1e4 * want) < 1e-9


def test_delayed_tone_phase_slope(oracle):
    T, C, N, P = 32, 64, 3, 1
    tau = np.array([0.0, 13e-9, 41e-9])
    f = np.arange(C) * (100e6 / C)
    ph = np.exp(-2j * np.pi * f[:, None] * tau[None, :])                      # [C, N]
    x = np.zeros((T, C, N, P, 2), dtype=np.float16)
    x[..., 0, 0] = ph.real
    x[..., 0, 1] = ph.imag
    V = oracle.xengine(x)
    for i in range(N):
        for j in range(i):
            v = V[:, oracle.baseline_index(i, j), 0, 0, 0] + 1j * V[:, oracle.baseline_index(i, j), 0, 0, 1]
            want = T * np.exp(+2j * np.pi * f * (tau[i] - tau[j]))
            assert np.max(np.abs(v - want)) < 2e-3 * T                        # fp16 quantisation of the tone
            slope = np.polyfit(f, np.unwrap(np.angle(v)), 1)[0] / (2 * np.pi)
            assert abs(slope - (tau[i] - tau[j])) < 0.02e-9


# ---- pin 8: additivity in time pins `accumulate` --------------------------------------------
def test_time_additivity_and_accumulate(oracle):
    rng = np.random.default_rng(8)
    T1, T2, C, N, P = 19, 30, 2, 5, 2
    x = rand_ci8(rng, T1 + T2, C, N, P)
    whole = oracle.xengine(x)
    acc = oracle.xengine(x[:T1])
    first = acc.copy()
    ret = oracle.xengine(x[T1:], accumulate_into=acc)
    assert ret is acc
    assert np.array_equal(acc, whole)
    assert np.array_equal(first + oracle.xengine(x[T1:]), whole)
    xf = rng.standard_normal((T1 + T2, C, N, P, 2)).astype(np.float16)
    wf = oracle.xengine(xf)
    af = oracle.xengine(xf[T1:], accumulate_into=oracle.xengine(xf[:T1]))
    assert np.max(np.abs(af - wf)) < 1e-12 * np.abs(wf).max()


# ---- pin 9: exact rotation by j, integer gain -----------------------------------------------
def test_rotation_and_gain(oracle):
    rng = np.random.default_rng(9)
    T, C, N, P = 25, 2, 4, 2
    x = rand_ci8(rng, T, C, N, P, -60, 60)
    k = 2
    y = x.copy()
    y[:, :, k, :, 0] = -x[:, :, k, :, 1]          # multiply station k by j: (re, im) -> (-im, re)
    y[:, :, k, :, 1] = x[:, :, k, :, 0]
    V, W = oracle.xengine(x), oracle.xengine(y)
    v = V[..., 0] + 1j * V[..., 1]
    w = W[..., 0] + 1j * W[..., 1]
    for i in range(N):
        for j in range(i + 1):
            b = oracle.baseline_index(i, j)
            if i == k and j == k:
                f = 1
            elif i == k:
                f = -1j            # conj(j x_k) x_j = -j V_kj
            elif j == k:
                f = 1j             # conj(x_i) (j x_k) = +j V_ik
            else:
                f = 1
            assert np.array_equal(w[:, b], f * v[:, b])
    g = 2
    assert np.array_equal(oracle.xengine((x * g).astype(np.int8)), g * g * V)


# ---- pin 10: beam-sum identity --------------------------------------------------------------
def test_beam_sum_identity(oracle):
    rng = np.random.default_rng(10)
    T, C, N, P = 41, 3, 7, 2
    x = rand_ci8(rng, T, C, N, P)
    V = oracle.xengine(x)
    xi = x.astype(np.int64)
    sr = xi[..., 0].sum(axis=(2, 3))
    si = xi[..., 1].sum(axis=(2, 3))
    beam = (sr * sr + si * si).sum(axis=0)                                     # [C]
    tot = np.zeros(C, dtype=np.int64)
    for i in range(N):
        for j in range(i + 1):
            re = V[:, oracle.baseline_index(i, j), :, :, 0].sum(axis=(1, 2))
            tot += re if i == j else 2 * re          # off-diagonal blocks count twice (H = H^H)
    assert np.array_equal(tot, beam)


# ---- pin 11: station permutation permutes the output ----------------------------------------
def test_station_permutation(oracle):
    rng = np.random.default_rng(11)
    T, C, N, P = 20, 2, 5, 2
    x = rand_ci8(rng, T, C, N, P)
    perm = np.array([3, 0, 4, 1, 2])
    V, W = oracle.xengine(x), oracle.xengine(x[:, :, perm])
    for i in range(N):
        for j in range(i + 1):
            a, b = perm[i], perm[j]
            w = W[:, oracle.baseline_index(i, j)]
            if a >= b:
                assert np.array_equal(w, V[:, oracle.baseline_index(a, b)])
            else:
                ref = V[:, oracle.baseline_index(b, a)].transpose(0, 2, 1, 3).copy()
                ref[..., 1] *= -1
                assert np.array_equal(w, ref)


# ---- channel selection and argument checks --------------------------------------------------
def test_channel_subset_and_threads(oracle):
    rng = np.random.default_rng(12)
    x = rand_ci8(rng, 16, 6, 3, 2)
    V = oracle.xengine(x)
    sel = [5, 0, 3]
    assert np.array_equal(oracle.xengine(x, chans=sel), V[sel])
    oracle.set_threads(1)
    assert np.array_equal(oracle.xengine(x), V)
    oracle.set_threads(oracle.max_threads())
    with pytest.raises(RuntimeError):
        oracle.xengine(x, chans=[6])
    with pytest.raises(TypeError):
        oracle.xengine(x.astype(np.int16))


def test_empty_time_gives_zeros(oracle):
    x = np.zeros((0, 2, 3, 2, 2), dtype=np.int8)
    assert not oracle.xengine(x).any()


# ---- the input recipe and the oracle agree on the expected sky phase (reading A13) ----------
def test_sky_delay_recipe_expected_phase(oracle):
    from paper_1305_5639_b200 import inputs
    cfg = dict(inputs.CONFIGS["cfg2"], N=6)
    T, C = 32768, 8      # noise in V ~ 1000 sqrt(T) = 2.8 % of the 200 T signal; 0.15 is > 5 sigma
    x = inputs.make_input(cfg, T=T, C=C).numpy()
    assert x.min() >= -127 and x.max() <= 127
    V = oracle.xengine(x)
    tau = inputs.station_delays(cfg["N"], cfg["seed"]).numpy()
    f = np.arange(C) * (inputs.BAND_HZ / C)
    for i in range(cfg["N"]):
        for j in range(i):
            b = oracle.baseline_index(i, j)
            for p in range(2):
                v = V[:, b, p, p, 0] + 1j * V[:, b, p, p, 1]
                want = 200.0 * T * np.exp(+2j * np.pi * f * (tau[i] - tau[j]))
                assert np.max(np.abs(v - want)) < 0.15 * 200.0 * T
            cross = V[:, b, 0, 1, 0] + 1j * V[:, b, 0, 1, 1]
            assert np.max(np.abs(cross)) < 0.15 * 200.0 * T
