"""Seeded synthetic channelised voltages for the X-engine (shared by tests, bench and smoke).

This module holds NONE of the method's arithmetic: it only synthesises telescope-like input
in the layout the boundary defines, ``x[T, C, N, P, 2]`` with the last axis (re, im), as
``torch.int8`` (ci8) or ``torch.float16`` (cf16).  Both the CUDA path and the CPU oracle consume
the SAME bytes (tests copy the tensor to the host for the oracle), so parity never depends on
the generator.  The recipes restate BASELINE.json's five configs;
they stand in for the paper's Fornax test streams, which were never
published.  Station delays are always drawn on the CPU so they do not depend on the device.
"""
import math

import torch

BAND_HZ = 100e6       # configs 2 and 4: "a linear phase across a 100 MHz band"
TAU_MAX_S = 50e-9     # "a random per-station delay in [0, 50] ns"


def _gen(seed, device):
    g = torch.Generator(device=device)
    g.manual_seed(int(seed))
    return g


def _t_chunk(C, N, P, budget_bytes=1 << 28):
    per_row = C * N * P * 2 * 4 * 3   # ~3 fp32 temporaries per element
    return max(1, budget_bytes // per_row)


def _quantise_ci8(v):
    """rint (ties-to-even) and clip to [-127, 127] -> int8; -128 is never produced."""
    return torch.clamp(torch.round(v), -127.0, 127.0).to(torch.int8)


def gauss_ci8(T, C, N, P, sigma, seed, device="cpu"):
    """Configs 1 and 5: re, im i.i.d. clip(rint(N(0, sigma^2)), +-127)."""
    g = _gen(seed, device)
    out = torch.empty((T, C, N, P, 2), dtype=torch.int8, device=device)
    step = _t_chunk(C, N, P)
    for t0 in range(0, T, step):
        t1 = min(T, t0 + step)
        v = torch.randn((t1 - t0, C, N, P, 2), generator=g, device=device, dtype=torch.float32)
        out[t0:t1] = _quantise_ci8(v * float(sigma))
    return out


def station_delays(N, seed):
    """tau_s ~ U[0, 50 ns], one per station, shared by both polarisations and all calls."""
    g = _gen(seed, "cpu")
    return torch.rand((N,), generator=g, dtype=torch.float64) * TAU_MAX_S


def sky_delay_ci8(T, C, N, P, seed, call=0, device="cpu", sigma_noise=20.0, sigma_sky=10.0):
    """Configs 2 and 4: x = n + g * exp(-j 2 pi f_c tau_s), rounded and clipped.

    n: independent noise, re/im ~ N(0, sigma_noise^2) per (t, c, s, p).
    g: common sky signal, re/im ~ N(0, sigma_sky^2) per (t, c, p), shared by all stations.
    f_c = c * BAND_HZ / C.  tau_s from ``station_delays(N, seed)`` (same for every call);
    n and g are fresh per ``call`` (data seed = seed * 1000 + call).
    """
    tau = station_delays(N, seed)
    f = torch.arange(C, dtype=torch.float64) * (BAND_HZ / C)
    phi = (2.0 * math.pi) * f[:, None] * tau[None, :]                 # [C, N]
    cs = torch.cos(phi).to(torch.float32).to(device)[None, :, :, None]
    sn = torch.sin(phi).to(torch.float32).to(device)[None, :, :, None]
    g = _gen(int(seed) * 1000 + int(call), device)
    out = torch.empty((T, C, N, P, 2), dtype=torch.int8, device=device)
    step = _t_chunk(C, N, P)
    for t0 in range(0, T, step):
        t1 = min(T, t0 + step)
        n = torch.randn((t1 - t0, C, N, P, 2), generator=g, device=device, dtype=torch.float32)
        sky = torch.randn((t1 - t0, C, 1, P, 2), generator=g, device=device, dtype=torch.float32)
        sky = sky * float(sigma_sky)
        gr, gi = sky[..., 0], sky[..., 1]
        v = n * float(sigma_noise)
        v[..., 0] += gr * cs + gi * sn          # Re g e^{-j phi}
        v[..., 1] += gi * cs - gr * sn          # Im g e^{-j phi}
        out[t0:t1] = _quantise_ci8(v)
    return out


def corr_phase_cf16(T, C, N, P, seed, device="cpu", amp=0.3):
    """Config 3: x = n + amp * e^{j phi_s} * g_p(t, c), rounded to fp16 (round-to-nearest).

    n, g: complex Gaussian, sigma = 1 per component; phi_s ~ U[0, 2 pi) per station.
    """
    gp = _gen(seed, "cpu")
    phi = torch.rand((N,), generator=gp, dtype=torch.float64) * (2.0 * math.pi)
    cs = torch.cos(phi).to(torch.float32).to(device)[None, None, :, None]
    sn = torch.sin(phi).to(torch.float32).to(device)[None, None, :, None]
    g = _gen(int(seed) * 1000, device)
    out = torch.empty((T, C, N, P, 2), dtype=torch.float16, device=device)
    step = _t_chunk(C, N, P)
    for t0 in range(0, T, step):
        t1 = min(T, t0 + step)
        v = torch.randn((t1 - t0, C, N, P, 2), generator=g, device=device, dtype=torch.float32)
        sky = torch.randn((t1 - t0, C, 1, P, 2), generator=g, device=device, dtype=torch.float32)
        gr, gi = sky[..., 0] * float(amp), sky[..., 1] * float(amp)
        v[..., 0] += gr * cs - gi * sn          # Re g e^{+j phi}
        v[..., 1] += gi * cs + gr * sn          # Im g e^{+j phi}
        out[t0:t1] = v.to(torch.float16)
    return out


# ---------------------------------------------------------------------------------------
# BASELINE.json's five configs.  "calls" > 1 means integration across successive
# corr_xengine calls (accumulate = 0, 1, 1, ...), each call on a fresh buffer.
# ---------------------------------------------------------------------------------------
CONFIGS = {
    "cfg1": dict(N=16, P=2, C=64, T=256, dtype="ci8", recipe="gauss", sigma=16.0, seed=1001, calls=1),
    "cfg2": dict(N=64, P=2, C=1024, T=1024, dtype="ci8", recipe="sky_delay", seed=1002, calls=1),
    "cfg3": dict(N=128, P=2, C=1024, T=4096, dtype="cf16", recipe="corr_phase", seed=1003, calls=1),
    "cfg4": dict(N=256, P=2, C=1024, T=2048, dtype="ci8", recipe="sky_delay", seed=1004, calls=4),
}
for _n in (32, 64, 128, 256, 512, 1024):
    CONFIGS["cfg5_n%d" % _n] = dict(N=_n, P=2, C=131072 // _n, T=2048, dtype="ci8", recipe="gauss",
                                    sigma=20.0, seed=1500 + int(math.log2(_n)), calls=1)


# the rectangle a space-division node processes: two groups of 256 dual-pol stations
# (N here is group A, Nb group B; group B is drawn with seed + 500), values as config 5.
CONFIGS["cross_n256"] = dict(N=256, Nb=256, P=2, C=512, T=2048, dtype="ci8", recipe="gauss", sigma=20.0, seed=1600, calls=1)


def make_input_b(cfg, call=0, device="cpu", T=None, C=None):
    """Group B of a cross workload (same recipe, Nb stations, its own seed)."""
    cfg_b = dict(cfg, N=cfg["Nb"], seed=cfg["seed"] + 500)
    return make_input(cfg_b, call, device, T, C)


def make_input(cfg, call=0, device="cpu", T=None, C=None):
    """Input tensor of one call of a config (dict from CONFIGS); T / C may be overridden to
    cut a smaller case of the same recipe (used by CPU-sized parity tests)."""
    T = cfg["T"] if T is None else T
    C = cfg["C"] if C is None else C
    N, P = cfg["N"], cfg["P"]
    r = cfg["recipe"]
    if r == "gauss":
        return gauss_ci8(T, C, N, P, cfg["sigma"], cfg["seed"] * 1000 + call, device)
    if r == "sky_delay":
        return sky_delay_ci8(T, C, N, P, cfg["seed"], call, device)
    if r == "corr_phase":
        return corr_phase_cf16(T, C, N, P, cfg["seed"] + call, device)
    raise ValueError("unknown recipe %r" % r)
