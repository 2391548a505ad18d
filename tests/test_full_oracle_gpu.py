"""Full-coverage parity of every BASELINE.json config point: EVERY channel, baseline and polarisation product of the GPU
result against the CPU oracle (the default suite samples channels of the big configs to stay within minutes).

Seven of the ten config points cost the oracle at most ~15 s each on the GPU box's host cores (config 1, 2, 3 and config 5
at N = 32 .. 256: about 40 s together) and run BY DEFAULT; config 4, N = 512 and N = 1024 (~2.3e12 complex MACs, minutes)
stay opt-in:

    CORR_FULL_ORACLE=1 python -m pytest tests/test_full_oracle_gpu.py -m gpu -q -s        # all ten config points
    CORR_FULL_ORACLE=cfg4 python -m pytest tests/test_full_oracle_gpu.py -m gpu -q -s     # the default seven + config 4
    CORR_FULL_ORACLE=0 ...                                                                 # none (skip them all)

int8 configs: bit-exact.  fp16 config: max over all visibilities of |dV| / sqrt(V_ii V_jj) <= 2e-5.
The last recorded run is profiles/r2b_full_oracle_parity.md.
"""
import os
import time

import numpy as np
import pytest
import torch

from paper_1305_5639_b200 import inputs

pytestmark = pytest.mark.gpu

ALL = ["cfg1", "cfg2", "cfg3", "cfg4"] + ["cfg5_n%d" % n for n in (32, 64, 128, 256, 512, 1024)]
DEFAULT = ["cfg1", "cfg2", "cfg3"] + ["cfg5_n%d" % n for n in (32, 64, 128, 256)]
_sel = os.environ.get("CORR_FULL_ORACLE", "")
SELECTED = ALL if _sel == "1" else [] if _sel == "0" else DEFAULT + [n for n in _sel.split(",") if n in ALL]


@pytest.mark.parametrize("name", ALL)
def test_full_coverage(oracle, name, capsys):
    if name not in SELECTED:
        pytest.skip("opt-in (minutes of oracle time): set CORR_FULL_ORACLE=1 or name it, e.g. CORR_FULL_ORACLE=%s" % name)
    from paper_1305_5639_b200 import binding
    cfg = inputs.CONFIGS[name]
    N, P, C, T, dtype, calls = cfg["N"], cfg["P"], cfg["C"], cfg["T"], cfg["dtype"], cfg["calls"]
    xs = [inputs.make_input(cfg, call=k, device="cuda") for k in range(calls)]
    with binding.Correlator(N, P, C, T, dtype) as h:
        out = None
        for k, x in enumerate(xs):
            out = h.xengine(x, out, accumulate=k > 0)
        torch.cuda.synchronize()
        kernel = h.kernel
    got = out.cpu().numpy()
    t0 = time.time()
    worst, bad, step = 0.0, 0, max(1, min(C, 64))
    auto_b = np.array([i * (i + 1) // 2 + i for i in range(N)])
    i_of_b = np.concatenate([np.full(i + 1, i) for i in range(N)])
    j_of_b = np.concatenate([np.arange(i + 1) for i in range(N)])
    for c0 in range(0, C, step):                       # oracle in channel slabs (bounded host memory)
        chans = list(range(c0, min(C, c0 + step)))
        want = None
        for x in xs:
            want = oracle.xengine(x[:, chans].contiguous().cpu().numpy(), accumulate_into=want)
        g = got[chans]
        if dtype == "ci8":
            bad += int((g.astype(np.int64) != want).sum())
        else:
            auto = np.stack([want[:, auto_b, p, p, 0] for p in range(P)], axis=-1)
            d = g.astype(np.float64) - want
            err = np.sqrt(d[..., 0] ** 2 + d[..., 1] ** 2) / np.sqrt(auto[:, i_of_b, :, None] * auto[:, j_of_b, None, :])
            worst = max(worst, float(err.max()))
    secs = time.time() - t0
    n_vis = C * (N * (N + 1) // 2) * P * P
    with capsys.disabled():          # the figures belong in the pytest output also without -s
        if dtype == "ci8":
            print("\n%s (%s kernel): %d visibilities x 2 words, all %d channels, %d call(s): %d mismatching words  [oracle %.0f s]"
                  % (name, kernel, n_vis, C, calls, bad, secs), flush=True)
        else:
            print("\n%s (%s kernel): %d visibilities, all %d channels: max normalised error %.3e (bar 2e-5)  [oracle %.0f s]"
                  % (name, kernel, n_vis, C, worst, secs), flush=True)
    if dtype == "ci8":
        assert bad == 0, "%s: %d mismatching words" % (name, bad)
    else:
        assert worst <= 2e-5
