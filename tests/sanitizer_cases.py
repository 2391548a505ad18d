#!/usr/bin/env python
"""Small geometries through EVERY kernel of libcorr.so, for `compute-sanitizer` (memcheck / racecheck / synccheck / initcheck).

    compute-sanitizer --tool memcheck  python tests/sanitizer_cases.py
    compute-sanitizer --tool racecheck python tests/sanitizer_cases.py
    compute-sanitizer --tool synccheck python tests/sanitizer_cases.py

Not collected by pytest (the sanitizers slow every launch by orders of magnitude); each case is also checked against the
oracle so a run proves the instrumented kernels still compute the right thing.  Results: profiles/r2_sanitizer.md.
"""
import os
import sys

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
from paper_1305_5639_b200 import binding, inputs      # noqa: E402
import oracle                                          # noqa: E402
from oracle import fengine as fo                       # noqa: E402


def exact(got, want, what):
    ok = bool((got.astype(np.int64) == want).all())
    print("%-60s %s" % (what, "ok" if ok else "MISMATCH"), flush=True)
    if not ok:
        raise SystemExit(1)


def main():
    torch.cuda.set_device(0)
    # triangle, every kernel variant, two calls (store + reduce-add); ragged tiles and T
    for kernel, (N, P, C, T) in [("single", (40, 2, 3, 200)), ("pair", (72, 2, 5, 300)), ("pair", (136, 2, 4, 260)),
                                 ("simt", (33, 2, 2, 50)), ("single", (24, 1, 2, 96)), ("pair", (256, 2, 3, 384))]:
        x = inputs.gauss_ci8(T, C, N, P, 40.0, seed=100 + N)
        with binding.Correlator(N, P, C, T, "ci8") as h:
            h.set_kernel(kernel)
            out = h.xengine(x.cuda())
            out = h.xengine(x.cuda(), out, accumulate=True)
            torch.cuda.synchronize()
        exact(out.cpu().numpy(), 2 * oracle.xengine(x.numpy()), "triangle ci8 %s N=%d P=%d C=%d T=%d" % (kernel, N, P, C, T))
    # fp16 (several TMEM passes folded by reduce-adds)
    for kernel, (N, P, C, T) in [("pair", (64, 2, 3, 2100)), ("single", (24, 2, 2, 1100))]:
        x = inputs.corr_phase_cf16(T, C, N, P, seed=200 + N)
        with binding.Correlator(N, P, C, T, "cf16") as h:
            h.set_kernel(kernel)
            out = h.xengine(x.cuda())
            torch.cuda.synchronize()
        want = oracle.xengine(x.numpy())
        err = np.abs(out.cpu().numpy() - want).max() / np.abs(want).max()
        print("%-60s %s (max |d| / max |V| = %.2e)" % ("triangle cf16 %s N=%d T=%d" % (kernel, N, T), "ok" if err < 1e-5 else "MISMATCH", err))
        if err >= 1e-5:
            raise SystemExit(1)
    # cross-only rectangle
    xa, xb = inputs.gauss_ci8(200, 3, 72, 2, 30.0, seed=5), inputs.gauss_ci8(200, 3, 136, 2, 30.0, seed=6)
    with binding.CrossCorrelator(72, 136, 2, 3, 200, "ci8") as h:
        out = h.xengine_cross(xa.cuda(), xb.cuda())
        out = h.xengine_cross(xa.cuda(), xb.cuda(), out, accumulate=True)
        torch.cuda.synchronize()
    exact(out.cpu().numpy(), 2 * oracle.xengine_cross(xa.numpy(), xb.numpy()), "cross ci8 72 x 136 stations")
    # short integrations, channel windows, host-buffer pipeline
    x = inputs.gauss_ci8(256, 6, 80, 2, 40.0, seed=7)
    with binding.Correlator(80, 2, 6, 256, "ci8") as h:
        got = h.xengine_dumps(x.cuda(), 4).cpu().numpy()
    for d in range(4):
        exact(got[d], oracle.xengine(x[d * 64:(d + 1) * 64].numpy()), "dumps ci8 N=80, integration %d of 4" % d)
    want = oracle.xengine(x.numpy())
    out = torch.zeros((6, 80 * 81 // 2, 2, 2, 2), dtype=torch.int32, device="cuda")
    for c0, n in [(0, 2), (2, 3), (5, 1)]:
        with binding.Correlator(80, 2, 6, 256, "ci8", window=(c0, n)) as h:
            h.xengine(x.cuda(), out)
    torch.cuda.synchronize()
    exact(out.cpu().numpy(), want, "three channel windows of one buffer")
    with binding.Correlator(80, 2, 6, 256, "ci8") as h:
        oh = torch.empty(h.output_shape(), dtype=torch.int32).pin_memory()
        h.xengine_host(x.pin_memory(), None)
        h.xengine_host(x.pin_memory(), oh, accumulate=True)
    exact(oh.numpy(), 2 * want, "corr_xengine_host pipeline (6 windows, 2 calls)")
    # corner turn
    with binding.Correlator(24, 2, 5, 100, "ci8") as h:
        xc = inputs.gauss_ci8(100, 5, 24, 2, 30.0, seed=8)
        ws = h.corner_turn(xc.cuda())
        torch.cuda.synchronize()
        planes = ws.cpu().view(torch.int8).view(2, 5, 48, h.workspace_time, 2)
    ref = xc.reshape(100, 5, 48, 2).permute(1, 2, 0, 3)
    print("%-60s %s" % ("corner turn ci8", "ok" if torch.equal(planes[0, :, :, :100], ref) else "MISMATCH"))
    # F-engine (fp16 and requantised int8 output)
    g = torch.Generator().manual_seed(9)
    s = torch.randint(-128, 128, (33, 5 * 256), generator=g, dtype=torch.int8)
    S = fo.fengine(s.numpy())
    got = binding.fengine(s.cuda()).cpu().numpy().astype(np.float64)
    err = np.abs(got[..., 0] + 1j * got[..., 1] - S).max()
    print("%-60s %s (max |d| = %.3f)" % ("F-engine fp16 33 streams x 5 spectra", "ok" if err < 16.5 else "MISMATCH", err))
    codes = binding.fengine(s.cuda(), scale=1.0 / 64).cpu().numpy()
    want_c, _ = fo.quantise_ci8(S, 1.0 / 64)
    print("%-60s %s" % ("F-engine int8 codes", "ok" if np.abs(codes.astype(int) - want_c).max() <= 1 else "MISMATCH"))
    print("all sanitizer cases done")


if __name__ == "__main__":
    main()
