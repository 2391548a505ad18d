"""CPU oracle for the corner-turn kernel (piece (a)) -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

The corner turn is pure data movement (the B200 analogue of the paper's "indexing ... for optimizing the
GPU memory access"), so its oracle is the definition written as plain loops over every sample:

    ws    [c][m][t] = in[t][c][m]                         m = s * P + p, complex kept as (re, im)
    ws_rot[c][m][t] = (im, -re) of the same sample        the plane a K-major imaginary-part product would read
    both zero for T <= t < Tp

The negation is done in a wider type and reported as such: for complex int8, re = -128 has no int8 negative; this
oracle returns int16 planes for int8 input, so the caller decides what the kernel's contract is there (include/corr.h:
the kernel saturates -(-128) to 127).  Only tests/ may import this module.
"""
import numpy as np


def corner_turn(x, Tp):
    """x [T, C, N, P, 2] int8 / float16 -> (ws, ws_rot), each [C, N*P, Tp, 2]; int16 for int8 input, else float16."""
    x = np.asarray(x)
    if x.ndim != 5 or x.shape[-1] != 2 or x.dtype not in (np.int8, np.float16):
        raise ValueError("x must be int8 or float16 [T, C, N, P, 2]")
    T, C, N, P, _ = x.shape
    if Tp < T:
        raise ValueError("Tp must be >= T")
    wide = np.int16 if x.dtype == np.int8 else np.float16
    ws = np.zeros((C, N * P, Tp, 2), dtype=wide)
    rot = np.zeros((C, N * P, Tp, 2), dtype=wide)
    for t in range(T):
        for c in range(C):
            for s in range(N):
                for p in range(P):
                    re, im = wide(x[t, c, s, p, 0]), wide(x[t, c, s, p, 1])
                    m = s * P + p
                    ws[c, m, t, 0], ws[c, m, t, 1] = re, im
                    rot[c, m, t, 0], rot[c, m, t, 1] = im, -re
    return ws, rot
