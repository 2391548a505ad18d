#!/usr/bin/env python
"""Full-coverage parity of a BASELINE.json config: EVERY channel, baseline and polarisation product of the GPU result
against the CPU oracle (the pytest suite samples channels of the big configs to stay within minutes).

    python tests/full_oracle_check.py cfg2 cfg3 cfg4 [cfg5_n512 ...]

int8 configs: bit-exact.  fp16 config: max over all visibilities of |dV| / sqrt(V_ii V_jj) <= 2e-5.
Takes minutes of host time for the large configs (config 4: 4.4e12 complex MACs on the host cores).
"""
import os
import sys
import time

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
from paper_1305_5639_b200 import binding, inputs      # noqa: E402
import oracle                                          # noqa: E402


def main(names):
    for name in names:
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
        for c0 in range(0, C, step):                       # oracle in channel slabs (bounded host memory)
            chans = list(range(c0, min(C, c0 + step)))
            want = None
            for x in xs:
                want = oracle.xengine(x[:, chans].contiguous().cpu().numpy(), accumulate_into=want)
            g = got[chans]
            if dtype == "ci8":
                bad += int((g.astype(np.int64) != want).sum())
            else:
                auto_b = np.array([i * (i + 1) // 2 + i for i in range(N)])
                i_of_b = np.concatenate([np.full(i + 1, i) for i in range(N)])
                j_of_b = np.concatenate([np.arange(i + 1) for i in range(N)])
                auto = np.stack([want[:, auto_b, p, p, 0] for p in range(P)], axis=-1)
                d = g.astype(np.float64) - want
                err = np.sqrt(d[..., 0] ** 2 + d[..., 1] ** 2) / np.sqrt(auto[:, i_of_b, :, None] * auto[:, j_of_b, None, :])
                worst = max(worst, float(err.max()))
        secs = time.time() - t0
        n_vis = C * (N * (N + 1) // 2) * P * P
        if dtype == "ci8":
            print("%s (%s kernel): %d visibilities x 2 words, all %d channels, %d call(s): %d mismatching words  [oracle %.0f s]"
                  % (name, kernel, n_vis, C, calls, bad, secs), flush=True)
            assert bad == 0
        else:
            print("%s (%s kernel): %d visibilities, all %d channels: max normalised error %.3e (bar 2e-5)  [oracle %.0f s]"
                  % (name, kernel, n_vis, C, worst, secs), flush=True)
            assert worst <= 2e-5


if __name__ == "__main__":
    main(sys.argv[1:] or ["cfg2"])
