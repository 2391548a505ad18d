"""Pins of the rectangular (cross-only) oracle, oracle.xengine_cross (Sec. 4: "a rectangle pattern
for cross-correlations only").  CPU only.  It is pinned to things other than itself: numpy complex128 einsum,
a library ZGEMM, the already pinned triangle oracle, the conjugate-swap identity, a closed form."""
import numpy as np
import pytest


def _rand_ci8(rng, T, C, N, P, lo=-127, hi=128):
    return rng.integers(lo, hi, size=(T, C, N, P, 2), dtype=np.int8)


def _cplx(x):
    return x[..., 0].astype(np.float64) + 1j * x[..., 1].astype(np.float64)


@pytest.mark.parametrize("Na,Nb,P,C,T", [(1, 1, 1, 1, 1), (2, 3, 2, 2, 5), (4, 1, 1, 3, 7), (3, 5, 2, 1, 9)])
def test_cross_bruteforce_einsum(oracle, Na, Nb, P, C, T):
    rng = np.random.default_rng(100 + Na * 7 + Nb)
    xa, xb = _rand_ci8(rng, T, C, Na, P), _rand_ci8(rng, T, C, Nb, P)
    V = oracle.xengine_cross(xa, xb)
    ref = np.einsum("tcip,tcjq->cijpq", np.conj(_cplx(xa)), _cplx(xb))      # exact: sums far below 2^53
    assert V.shape == (C, Na, Nb, P, P, 2) and V.dtype == np.int64
    assert (V[..., 0] == np.rint(ref.real).astype(np.int64)).all()
    assert (V[..., 1] == np.rint(ref.imag).astype(np.int64)).all()


def test_cross_reduces_to_zgemm(oracle):
    rng = np.random.default_rng(7)
    T, C, Na, Nb, P = 64, 2, 6, 9, 2
    xa, xb = _rand_ci8(rng, T, C, Na, P), _rand_ci8(rng, T, C, Nb, P)
    V = oracle.xengine_cross(xa, xb)
    for c in range(C):
        A = _cplx(xa)[:, c].reshape(T, Na * P)
        B = _cplx(xb)[:, c].reshape(T, Nb * P)
        H = (A.conj().T @ B).reshape(Na, P, Nb, P).transpose(0, 2, 1, 3)     # [i][j][p][q]
        assert (V[c, ..., 0] == np.rint(H.real)).all() and (V[c, ..., 1] == np.rint(H.imag)).all()


def test_cross_equals_the_off_diagonal_block_of_the_triangle(oracle):
    """Split N stations into B = stations [0, k) and A = stations [k, N): the rectangle A x B is exactly the
    triangle's rows i >= k, columns j < k (same conjugated side, same polarisation order)."""
    rng = np.random.default_rng(11)
    T, C, N, P, k = 33, 3, 7, 2, 3
    x = _rand_ci8(rng, T, C, N, P)
    tri = oracle.xengine(x)
    V = oracle.xengine_cross(np.ascontiguousarray(x[:, :, k:]), np.ascontiguousarray(x[:, :, :k]))
    for i in range(k, N):
        for j in range(k):
            assert (V[:, i - k, j] == tri[:, oracle.baseline_index(i, j)]).all()


def test_cross_conjugate_swap(oracle):
    rng = np.random.default_rng(13)
    T, C, Na, Nb, P = 20, 2, 4, 5, 2
    xa, xb = _rand_ci8(rng, T, C, Na, P), _rand_ci8(rng, T, C, Nb, P)
    V, W = oracle.xengine_cross(xa, xb), oracle.xengine_cross(xb, xa)
    Wt = W.transpose(0, 2, 1, 4, 3, 5)                    # [c][i][j][p][q] <- W[c][j][i][q][p]
    assert (V[..., 0] == Wt[..., 0]).all() and (V[..., 1] == -Wt[..., 1]).all()


def test_cross_constant_closed_form_and_accumulate(oracle):
    """xa == a_i, xb == b_j constant in time  =>  V_ij = T conj(a_i) b_j (asymmetric constants pin the sign of
    Im and which group is conjugated); integrating the block twice doubles it."""
    T, C, P = 10, 1, 1
    a = np.array([3 + 4j, -2 + 7j]); b = np.array([5 - 1j, 1 + 2j, -6 - 3j])
    xa = np.zeros((T, C, 2, P, 2), np.int8); xb = np.zeros((T, C, 3, P, 2), np.int8)
    xa[..., 0], xa[..., 1] = a.real[None, None, :, None], a.imag[None, None, :, None]
    xb[..., 0], xb[..., 1] = b.real[None, None, :, None], b.imag[None, None, :, None]
    V = oracle.xengine_cross(xa, xb)
    want = T * np.conj(a)[:, None] * b[None, :]
    assert (V[0, :, :, 0, 0, 0] == want.real).all() and (V[0, :, :, 0, 0, 1] == want.imag).all()
    V2 = oracle.xengine_cross(xa, xb, accumulate_into=V.copy())
    assert (V2 == 2 * V).all()


def test_cross_cf16_against_zgemm_and_channel_subset(oracle):
    rng = np.random.default_rng(17)
    T, C, Na, Nb, P = 48, 4, 3, 4, 2
    xa = rng.standard_normal((T, C, Na, P, 2)).astype(np.float16)
    xb = rng.standard_normal((T, C, Nb, P, 2)).astype(np.float16)
    V = oracle.xengine_cross(xa, xb, chans=[3, 1])
    assert V.shape[0] == 2 and V.dtype == np.float64
    for k, c in enumerate([3, 1]):
        A = _cplx(xa)[:, c].reshape(T, Na * P); B = _cplx(xb)[:, c].reshape(T, Nb * P)
        H = (A.conj().T @ B).reshape(Na, P, Nb, P).transpose(0, 2, 1, 3)
        assert np.allclose(V[k, ..., 0], H.real, rtol=0, atol=1e-9) and np.allclose(V[k, ..., 1], H.imag, rtol=0, atol=1e-9)
