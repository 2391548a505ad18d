"""Pins for oracle/corner_turn.py (CPU only): a hand-written example, the library transpose, and the (im, -re) plane as a
multiplication by -j in complex arithmetic."""
import numpy as np
import pytest

from oracle import corner_turn as oc


def test_hand_example():
    # T = 2, C = 1, N = 2, P = 1: samples x[t][s] = (re, im)
    x = np.array([[[[[1, 2]], [[3, -4]]]], [[[[-5, 6]], [[-128, 127]]]]], dtype=np.int8)        # [2, 1, 2, 1, 2]
    ws, rot = oc.corner_turn(x, 3)
    assert ws.dtype == np.int16 and ws.shape == (1, 2, 3, 2)
    assert ws[0, 0].tolist() == [[1, 2], [-5, 6], [0, 0]]            # stream 0 over time, zero padded
    assert ws[0, 1].tolist() == [[3, -4], [-128, 127], [0, 0]]
    assert rot[0, 0].tolist() == [[2, -1], [6, 5], [0, 0]]
    assert rot[0, 1].tolist() == [[-4, -3], [127, 128], [0, 0]]      # -(-128) = 128 needs the wider type


@pytest.mark.parametrize("dtype", [np.int8, np.float16])
def test_equals_library_transpose_and_times_minus_j(dtype):
    rng = np.random.default_rng(5)
    T, C, N, P, Tp = 7, 3, 4, 2, 8
    x = (rng.integers(-128, 128, size=(T, C, N, P, 2)).astype(dtype) if dtype == np.int8
         else rng.standard_normal((T, C, N, P, 2)).astype(dtype))
    ws, rot = oc.corner_turn(x, Tp)
    ref = np.transpose(x.reshape(T, C, N * P, 2), (1, 2, 0, 3)).astype(ws.dtype)
    assert np.array_equal(ws[:, :, :T], ref) and not ws[:, :, T:].any() and not rot[:, :, T:].any()
    z = ws[..., 0].astype(np.float64) + 1j * ws[..., 1].astype(np.float64)
    zr = rot[..., 0].astype(np.float64) + 1j * rot[..., 1].astype(np.float64)
    assert np.array_equal(zr, -1j * z)                               # (im, -re) = -j (re + j im)


def test_rejects_bad_input():
    with pytest.raises(ValueError):
        oc.corner_turn(np.zeros((2, 1, 1, 1, 2), np.int16), 2)
    with pytest.raises(ValueError):
        oc.corner_turn(np.zeros((4, 1, 1, 1, 2), np.int8), 3)
