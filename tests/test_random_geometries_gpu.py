"""Randomised geometries (fixed seed): every mode (triangle, cross-only rectangle, short integrations) and every kernel
variant against the oracle, bit-exact on the int8 path, two calls each (store, then accumulate where the mode has it).
Covers ragged tiles, single-station problems, odd stream counts (SIMT), T below one pipeline stage."""
import numpy as np
import pytest
import torch

from paper_1305_5639_b200 import inputs

pytestmark = pytest.mark.gpu


def _cases(seed, n):
    rng = np.random.default_rng(seed)
    out = []
    for it in range(n):
        P = int(rng.choice([1, 2])); N = int(rng.integers(1, 300)); C = int(rng.integers(1, 5)); T = int(rng.integers(1, 600))
        mode = str(rng.choice(["herk", "cross", "dumps"]))
        kern = str(rng.choice(["auto", "pair", "single", "simt"]))
        Nb = int(rng.integers(1, 200))
        nd = int(rng.choice([d for d in range(1, 9) if T % d == 0]))
        out.append((mode, kern, N, Nb, P, C, T, nd, it))
    return out


@pytest.mark.parametrize("mode,kern,N,Nb,P,C,T,nd,it", _cases(20260101, 36))
def test_random_geometry_ci8(oracle, mode, kern, N, Nb, P, C, T, nd, it):
    from paper_1305_5639_b200 import binding
    x = inputs.gauss_ci8(T, C, N, P, 50.0, seed=8000 + it)
    if mode == "cross":
        xb = inputs.gauss_ci8(T, C, Nb, P, 50.0, seed=9000 + it)
        with binding.CrossCorrelator(N, Nb, P, C, T, "ci8") as h:
            got = h.xengine_cross(x.cuda(), xb.cuda())
            got = h.xengine_cross(x.cuda(), xb.cuda(), got, accumulate=True).cpu().numpy()
        want = 2 * oracle.xengine_cross(x.numpy(), xb.numpy())
    elif mode == "dumps":
        with binding.Correlator(N, P, C, T, "ci8") as h:
            got = h.xengine_dumps(x.cuda(), nd).cpu().numpy()
        Ts = T // nd
        want = np.stack([oracle.xengine(x[d * Ts:(d + 1) * Ts].numpy()) for d in range(nd)])
    else:
        with binding.Correlator(N, P, C, T, "ci8") as h:
            if kern != "auto" and (h.uses_tensor_cores or kern == "simt"):
                h.set_kernel(kern)
            got = h.xengine(x.cuda())
            got = h.xengine(x.cuda(), got, accumulate=True).cpu().numpy()
        want = 2 * oracle.xengine(x.numpy())
    torch.cuda.synchronize()
    assert got.shape == want.shape
    assert (got.astype(np.int64) == want).all()
