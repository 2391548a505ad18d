"""GPU parity: libcorr.so (through its C ABI, via the ctypes binding) against the CPU oracle.

Bar (BASELINE.json north_star): complex int8 -> int32 path BIT-EXACT, every word of the packed
output; complex fp16 -> fp32 path |dV_ij| <= 2e-5 * sqrt(V_ii^{pp} V_jj^{qq}) with both
autocorrelations taken from the fp64 oracle.  Small cases are compared element by element on all
channels; BASELINE.json's full-size configs are compared on sampled channels (every baseline and
polarisation product of each sampled channel) plus two identities that hold at any size on EVERY
channel: the beam-sum identity and real, non-negative autocorrelations.
"""
import numpy as np
import pytest
import torch

from paper_1305_5639_b200 import inputs

pytestmark = pytest.mark.gpu

FP16_TOL = 2e-5          # north_star: |dV_ij| <= 2e-5 * sqrt(V_ii * V_jj)


@pytest.fixture(scope="module")
def corr():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (there is no CPU fallback)")
    from paper_1305_5639_b200 import binding
    binding.lib()
    return binding


def run_gpu(corr, xs, dtype, accumulate_calls=True, host=False, kernel=None):
    """xs: list of input tensors (one per call).  Returns the int32/fp32 output as numpy."""
    T, C, N, P, _ = xs[0].shape
    with corr.Correlator(N, P, C, T, dtype) as h:
        if kernel is not None:
            h.set_kernel(kernel)
            assert h.kernel == kernel
        if host:
            out = torch.empty(h.output_shape(), dtype=torch.int32 if dtype == "ci8" else torch.float32)
            for k, x in enumerate(xs):
                h.xengine_host(x.cpu().contiguous(), out, accumulate=(k > 0 and accumulate_calls))
            return out.numpy(), h.uses_tensor_cores
        out = None
        for k, x in enumerate(xs):
            out = h.xengine(x.cuda(), out, accumulate=(k > 0 and accumulate_calls))
        torch.cuda.synchronize()
        return out.cpu().numpy(), h.uses_tensor_cores


def run_oracle(oracle, xs, chans=None):
    V = None
    for x in xs:
        V = oracle.xengine(x.cpu().numpy(), chans=chans, accumulate_into=V)
    return V


def assert_bit_exact(got, want):
    assert got.dtype == np.int32 and want.dtype == np.int64
    assert np.abs(want).max() < 2 ** 31
    bad = np.argwhere(got.astype(np.int64) != want)
    assert bad.size == 0, "first mismatches (c,b,p,q,reim): %s" % bad[:8].tolist()


def fp16_normalised_error(got, want, N, P):
    """max over all visibilities of |dV| / sqrt(V_ii^pp V_jj^qq) (autocorrelations from the oracle)."""
    i_of_b = np.concatenate([np.full(i + 1, i) for i in range(N)])
    j_of_b = np.concatenate([np.arange(i + 1) for i in range(N)])
    auto_b = np.array([i * (i + 1) // 2 + i for i in range(N)])
    auto = np.stack([want[:, auto_b, p, p, 0] for p in range(P)], axis=-1)        # [C, N, P]
    d = got.astype(np.float64) - want
    err = np.sqrt(d[..., 0] ** 2 + d[..., 1] ** 2)                                # [C, B, P, P]
    norm = np.sqrt(auto[:, i_of_b, :, None] * auto[:, j_of_b, None, :])
    return float((err / norm).max())


# ---------------------------------------------------------------------------------------------
# small cases: every channel, every word
# ---------------------------------------------------------------------------------------------
SMALL_CI8 = [
    # N, P, C, T      what it exercises
    (16, 2, 64, 256),   # BASELINE config 1
    (1, 1, 1, 1),       # smallest possible problem (SIMT path: row pitch not a multiple of 16 B)
    (1, 2, 3, 5),
    (4, 2, 5, 70),      # one partial tile, ragged T (not a multiple of the 64-sample stage)
    (8, 1, 3, 33),      # single polarisation on the tensor-core path
    (33, 2, 3, 100),    # N*P*2 = 132 B row: SIMT path
    (36, 2, 3, 130),    # 144 columns: two row blocks, ragged column cut
    (40, 1, 2, 64),
    (72, 2, 2, 192),    # 288 columns: >1 column block
    (100, 2, 2, 96),    # 400 columns: several row blocks + triangular cut + channel edge
    (130, 2, 1, 64),    # 520 columns
    (64, 2, 7, 1),      # T = 1
]


@pytest.mark.parametrize("N,P,C,T", SMALL_CI8)
def test_ci8_bit_exact_small(corr, oracle, N, P, C, T):
    x = inputs.gauss_ci8(T, C, N, P, 40.0, seed=7000 + N * 3 + T)
    got, tc = run_gpu(corr, [x], "ci8")
    assert tc == ((N * P * 2) % 16 == 0)
    assert_bit_exact(got, run_oracle(oracle, [x]))


# every tensor-core kernel variant on geometries that span ragged pair tiles, several row / column blocks,
# ragged T and both polarisation counts
KERNEL_CASES = [(16, 2, 5, 100), (64, 2, 9, 200), (72, 2, 3, 130), (96, 2, 4, 64), (128, 2, 5, 257),
                (136, 1, 3, 96), (200, 2, 2, 128), (256, 2, 3, 192), (320, 2, 2, 64)]


@pytest.mark.parametrize("kernel", ["single", "pair", "simt"])
@pytest.mark.parametrize("N,P,C,T", KERNEL_CASES)
def test_ci8_bit_exact_every_kernel(corr, oracle, kernel, N, P, C, T):
    x = inputs.gauss_ci8(T, C, N, P, 40.0, seed=7100 + N + T)
    got, _ = run_gpu(corr, [x, x], "ci8", kernel=kernel)          # two calls: store, then reduce-add
    want = run_oracle(oracle, [x, x])
    assert_bit_exact(got, want)


@pytest.mark.parametrize("kernel", ["single", "pair", "simt"])
@pytest.mark.parametrize("N,P,C,T", [(24, 2, 3, 100), (64, 2, 3, 1100), (96, 1, 2, 64), (160, 2, 2, 2100)])
def test_cf16_within_tolerance_every_kernel(corr, oracle, kernel, N, P, C, T):
    x = inputs.corr_phase_cf16(T, C, N, P, seed=7200 + N)
    got, _ = run_gpu(corr, [x], "cf16", kernel=kernel)
    err = fp16_normalised_error(got, run_oracle(oracle, [x]), N, P)
    assert err <= FP16_TOL, "normalised error %.3g" % err


def test_ci8_full_range_including_minus_128(corr, oracle):
    """-128 is exact on the direct (no-negation) feed: corr.h 'any value in [-128, 127] is exact'."""
    g = torch.Generator().manual_seed(11)
    x = torch.randint(-128, 128, (96, 3, 24, 2, 2), generator=g, dtype=torch.int8)
    x[0, 0] = -128
    x[1, 1] = 127
    got, tc = run_gpu(corr, [x], "ci8")
    assert tc
    assert_bit_exact(got, run_oracle(oracle, [x]))


def test_ci8_extreme_constant_fills_int32_range(corr, oracle):
    """All samples -128-128j for T = 65535: |V| = 2 * 128^2 * 65535 = 2^31 - 32768, the largest exact sum."""
    x = torch.full((4096, 1, 8, 2, 2), -128, dtype=torch.int8)
    with corr.Correlator(8, 2, 1, 4096, "ci8") as h:
        xd = x.cuda()
        out = h.xengine(xd)
        for _ in range(14):
            h.xengine(xd, out, accumulate=True)
        torch.cuda.synchronize()
        # 15 * 4096 = 61440 samples so far; 65535 is not a multiple of 4096, so stop here and check
        got = out.cpu().numpy()
        assert (got[..., 0] == 2 * 128 * 128 * 61440).all() and (got[..., 1] == 0).all()
        # one more call would be 65536 samples > 65535: refused, nothing launched
        with pytest.raises(corr.CorrError) as e:
            h.xengine(xd, out, accumulate=True)
        assert e.value.code == corr.CORR_EOVERFLOW
        torch.cuda.synchronize()
        assert (out.cpu().numpy() == got).all()


@pytest.mark.parametrize("host", [False, True])
def test_ci8_accumulate_across_calls(corr, oracle, host):
    """Integration across successive calls: accumulate = 0, 1, 1 equals the oracle's sum."""
    xs = [inputs.gauss_ci8(128, 4, 40, 2, 30.0, seed=7100 + k) for k in range(3)]
    got, _ = run_gpu(corr, xs, "ci8", host=host)
    assert_bit_exact(got, run_oracle(oracle, xs))
    # and concatenating the calls' samples is the same thing (additivity in time)
    assert_bit_exact(got, run_oracle(oracle, [torch.cat(xs, dim=0)]))


def test_accumulate_zero_overwrites_garbage(corr, oracle):
    x = inputs.gauss_ci8(64, 2, 20, 2, 30.0, seed=7200)
    with corr.Correlator(20, 2, 2, 64, "ci8") as h:
        out = torch.full(h.output_shape(), 0x5a5a5a5a, dtype=torch.int32, device="cuda")
        h.xengine(x.cuda(), out, accumulate=False)
        torch.cuda.synchronize()
        assert_bit_exact(out.cpu().numpy(), run_oracle(oracle, [x]))


def test_does_not_write_outside_the_output(corr):
    x = inputs.gauss_ci8(64, 3, 36, 2, 30.0, seed=7300).cuda()
    with corr.Correlator(36, 2, 3, 64, "ci8") as h:
        n = h.output_bytes // 4
        buf = torch.full((n + 2048,), 0x7e7e7e7e, dtype=torch.int32, device="cuda")
        out = buf[1024:1024 + n].view(h.output_shape())
        h.xengine(x, out)
        torch.cuda.synchronize()
        assert (buf[:1024] == 0x7e7e7e7e).all() and (buf[1024 + n:] == 0x7e7e7e7e).all()


def test_argument_errors(corr):
    with corr.Correlator(16, 2, 4, 64, "ci8") as h:
        x = torch.zeros(h.input_shape(), dtype=torch.int8, device="cuda")
        out = h.empty_output()
        L = corr.lib()
        assert L.corr_xengine(h._h, None, out.data_ptr(), 0, None) == corr.CORR_EINVAL
        assert L.corr_xengine(h._h, x.data_ptr(), None, 0, None) == corr.CORR_EINVAL
        assert L.corr_xengine(h._h, x.data_ptr() + 2, out.data_ptr(), 0, None) == corr.CORR_EINVAL
        assert b"aligned" in L.corr_last_error(h._h)
        assert h.input_bytes == x.numel() and h.output_bytes == out.numel() * 4


SMALL_CF16 = [(16, 2, 8, 256), (2, 2, 3, 40), (3, 1, 2, 17), (20, 2, 3, 100), (68, 2, 2, 160), (128, 2, 2, 512)]


@pytest.mark.parametrize("N,P,C,T", SMALL_CF16)
def test_cf16_within_tolerance_small(corr, oracle, N, P, C, T):
    x = inputs.corr_phase_cf16(T, C, N, P, seed=7400 + N)
    got, tc = run_gpu(corr, [x], "cf16")
    assert tc == ((N * P * 4) % 16 == 0)
    want = run_oracle(oracle, [x])
    assert fp16_normalised_error(got, want, N, P) <= FP16_TOL


def test_cf16_accumulate_across_calls(corr, oracle):
    xs = [inputs.corr_phase_cf16(256, 3, 24, 2, seed=7500 + k) for k in range(3)]
    got, _ = run_gpu(corr, xs, "cf16")
    assert fp16_normalised_error(got, run_oracle(oracle, xs), 24, 2) <= FP16_TOL


def test_stream_argument_is_honoured(corr, oracle):
    x = inputs.gauss_ci8(64, 4, 16, 2, 30.0, seed=7600)
    s = torch.cuda.Stream()
    with corr.Correlator(16, 2, 4, 64, "ci8") as h:
        with torch.cuda.stream(s):
            xd = x.cuda(non_blocking=False)
            out = h.xengine(xd, stream=s)
        s.synchronize()
        assert_bit_exact(out.cpu().numpy(), run_oracle(oracle, [x]))
        assert h.last_launch_count >= 1


def test_corner_turn_kernel(corr):
    """Piece (a): ws[c][m][t] = in[t][c][m], ws_rot = (im, -re), time zero-padded -- against oracle.corner_turn (plain
    loops, pinned in tests/test_oracle_corner_turn_pins.py).  The int8 case carries -128: the rotated plane saturates
    -(-128) to +127 (corr.h), everything else is exact."""
    from oracle import corner_turn as oc
    for dtype, N, P, C, T in [("ci8", 24, 2, 5, 100), ("ci8", 64, 2, 3, 256), ("cf16", 20, 2, 3, 70)]:
        if dtype == "ci8":
            x = inputs.gauss_ci8(T, C, N, P, 30.0, seed=7700)
            x[0, 0, 0, 0, 0] = -128
            x[T - 1, C - 1, N - 1, P - 1] = -128
        else:
            x = inputs.corr_phase_cf16(T, C, N, P, seed=7701)
        with corr.Correlator(N, P, C, T, dtype) as h:
            ws = h.corner_turn(x.cuda())
            torch.cuda.synchronize()
            Tp = h.workspace_time
            planes = ws.cpu().view(torch.int8 if dtype == "ci8" else torch.float16).view(2, C, N * P, Tp, 2).numpy()
        want_ws, want_rot = oc.corner_turn(x.numpy(), Tp)
        if dtype == "ci8":
            assert (want_rot == 128).sum() == 2                      # the two re = -128 samples
            want_rot = np.minimum(want_rot, 127)
        assert np.array_equal(planes[0].astype(want_ws.dtype), want_ws)
        assert np.array_equal(planes[1].astype(want_rot.dtype), want_rot)
        # one plane only (corr_corner_turn_planes): the first half of the workspace, nothing beyond it
        with corr.Correlator(N, P, C, T, dtype) as h:
            half = h.workspace_bytes // 2
            buf = torch.full((half + 4096,), 0x5a, dtype=torch.uint8, device="cuda")
            h.corner_turn(x.cuda(), buf[:half], planes=1)
            torch.cuda.synchronize()
            one = buf[:half].cpu().view(torch.int8 if dtype == "ci8" else torch.float16).view(C, N * P, Tp, 2).numpy()
            assert np.array_equal(one.astype(want_ws.dtype), want_ws) and (buf[half:] == 0x5a).all()


# ---------------------------------------------------------------------------------------------
# BASELINE.json configs at full size, in the launch configuration bench.py times
# ---------------------------------------------------------------------------------------------
def sample_channels(C, n, seed):
    rng = np.random.default_rng(seed)
    mid = rng.choice(np.arange(1, C - 1), size=min(n, C) - 2, replace=False) if C > 2 else []
    return np.unique(np.concatenate([[0, C - 1], mid]).astype(np.int32))


def beam_sum_identity(xs, got, N, P):
    """Both sides of  sum_{m,n} H_c[m][n] = sum_t |sum_m x[t][c][m]|^2  for EVERY channel (SURVEY pin 10).
    The right side is formed from the device-resident inputs in chunks of time with torch ops (exact in
    int64 for ci8, fp64 for cf16); the left side expands the packed triangle by Hermitian symmetry."""
    C = got.shape[0]
    integer = got.dtype == np.int32
    wide = torch.int64 if integer else torch.float64
    rhs = torch.zeros(C, dtype=wide, device=xs[0].device)
    for x in xs:
        for t0 in range(0, x.shape[0], 64):
            s = x[t0:t0 + 64].to(torch.int32 if integer else torch.float64).sum(dim=(2, 3)).to(wide)   # [t, C, 2]
            rhs += (s * s).sum(dim=(0, 2))
    g = torch.from_numpy(got)
    re = g[..., 0].to(wide)
    auto_b = torch.tensor([i * (i + 1) // 2 + i for i in range(N)])
    lhs = 2 * re.sum(dim=(1, 2, 3)) - re[:, auto_b].sum(dim=(1, 2, 3))            # cross terms twice, autos once
    return lhs.numpy(), rhs.cpu().numpy()


def check_full_config(corr, oracle, name, n_chan_sample):
    cfg = inputs.CONFIGS[name]
    N, P, C, T, dtype = cfg["N"], cfg["P"], cfg["C"], cfg["T"], cfg["dtype"]
    xs = [inputs.make_input(cfg, call=k, device="cuda") for k in range(cfg["calls"])]
    with corr.Correlator(N, P, C, T, dtype) as h:
        assert h.uses_tensor_cores
        out = None
        for k, x in enumerate(xs):
            out = h.xengine(x, out, accumulate=k > 0)
        torch.cuda.synchronize()
    got = out.cpu().numpy()
    chans = sample_channels(C, n_chan_sample, cfg["seed"])
    want = None
    for x in xs:
        want = oracle.xengine(x.cpu().numpy(), chans=chans, accumulate_into=want)
    lhs, rhs = beam_sum_identity(xs, got, N, P)
    auto_b = np.array([i * (i + 1) // 2 + i for i in range(N)])
    if dtype == "ci8":
        assert_bit_exact(got[chans], want)
        assert (lhs == rhs).all()
        for p in range(P):
            assert (got[:, auto_b, p, p, 1] == 0).all() and (got[:, auto_b, p, p, 0] >= 0).all()
    else:
        err = fp16_normalised_error(got[chans], want, N, P)
        assert err <= FP16_TOL, err
        # the per-visibility tolerance implies |lhs - rhs| <= tol * (sum_m sqrt(H_mm))^2
        autos = np.stack([got[:, auto_b, p, p, 0] for p in range(P)], axis=-1).astype(np.float64)   # [C, N, P]
        assert (autos > 0).all()
        bound = FP16_TOL * np.sqrt(autos).sum(axis=(1, 2)) ** 2
        assert (np.abs(lhs - rhs) <= bound).all()
        for p in range(P):
            assert (np.abs(got[:, auto_b, p, p, 1]) <= FP16_TOL * got[:, auto_b, p, p, 0]).all()


def test_config2_full_size(corr, oracle):
    check_full_config(corr, oracle, "cfg2", 24)


def test_config3_full_size_fp16(corr, oracle):
    check_full_config(corr, oracle, "cfg3", 8)


def test_config4_full_size_four_calls(corr, oracle):
    check_full_config(corr, oracle, "cfg4", 8)


def test_config1_own_recipe_every_word(corr, oracle):
    """BASELINE.json config 1 with its own recipe (sigma 16, seed 1001): every word of all 64 channels."""
    cfg = inputs.CONFIGS["cfg1"]
    x = inputs.make_input(cfg)
    got, tc = run_gpu(corr, [x], "ci8")
    assert tc and got.shape == (64, 136, 2, 2, 2)
    assert_bit_exact(got, run_oracle(oracle, [x]))


@pytest.mark.parametrize("N", [32, 64, 128, 256, 512, 1024])
def test_config5_sweep_points(corr, oracle, N):
    check_full_config(corr, oracle, "cfg5_n%d" % N, 4 if N <= 128 else 2)


# ---------------------------------------------------------------------------------------------
# channel windows (corr_create_window): windows of ONE input into ONE output
# ---------------------------------------------------------------------------------------------
def _windows(C, world):
    from paper_1305_5639_b200.shard import channel_range
    return [channel_range(C, world, r) for r in range(world)]


@pytest.mark.parametrize("world", [2, 3, 8])
@pytest.mark.parametrize("N,P,C,T,dtype,kernel", [(72, 2, 11, 200, "ci8", "pair"), (40, 2, 9, 130, "ci8", "single"),
                                                  (33, 2, 8, 50, "ci8", "simt"), (136, 1, 10, 96, "ci8", None),
                                                  (64, 2, 9, 1100, "cf16", None)])
def test_channel_windows_equal_the_unsharded_launch(corr, oracle, world, N, P, C, T, dtype, kernel):
    """`world` window plans over one [T][C][N][P] buffer, each writing its own slabs of one output (two calls: store, then
    accumulate): word for word the unsharded launch, and the oracle; a canary value in a window's foreign slabs survives."""
    x = (inputs.gauss_ci8(T, C, N, P, 40.0, seed=7900 + N) if dtype == "ci8" else inputs.corr_phase_cf16(T, C, N, P, seed=7900 + N))
    xd = x.cuda()
    with corr.Correlator(N, P, C, T, dtype) as h:
        if kernel:
            h.set_kernel(kernel)
        whole = h.xengine(xd)
        whole = h.xengine(xd, whole, accumulate=True)
        torch.cuda.synchronize()
    canary = 0x5a5a5a5a if dtype == "ci8" else 12345.0
    out = torch.full_like(whole, canary)
    for c0, c1 in _windows(C, world):
        if c1 == c0:
            continue
        with corr.Correlator(N, P, C, T, dtype, window=(c0, c1 - c0)) as hw:
            if kernel:
                hw.set_kernel(kernel)
            assert hw.input_bytes == xd.numel() * xd.element_size() and hw.output_bytes == out.numel() * 4
            before = out.clone()
            hw.xengine(xd, out)
            hw.xengine(xd, out, accumulate=True)
            torch.cuda.synchronize()
            keep = torch.ones(C, dtype=torch.bool, device="cuda"); keep[c0:c1] = False
            assert torch.equal(out[keep], before[keep])              # nothing outside the window's slabs was touched
    assert torch.equal(out, whole)                                   # word for word (also fp32: same kernel, same order)
    want = oracle.xengine(x.numpy())
    if dtype == "ci8":
        assert_bit_exact(out.cpu().numpy(), 2 * want)
    else:
        assert fp16_normalised_error(out.cpu().numpy(), 2 * want, N, P) <= FP16_TOL


def test_channel_windows_dumps_and_host_path(corr, oracle):
    """A window plan through corr_xengine_dumps and corr_xengine_host: only the window's columns / slabs are used."""
    N, P, C, T = 48, 2, 7, 192
    x = inputs.gauss_ci8(T, C, N, P, 40.0, seed=7950)
    want = oracle.xengine(x.numpy())
    c0, n = 2, 3
    with corr.Correlator(N, P, C, T, "ci8", window=(c0, n)) as h:
        out = torch.full((4,) + tuple(h.output_shape()), 77, dtype=torch.int32, device="cuda")
        h.xengine_dumps(x.cuda(), 4, out)
        torch.cuda.synchronize()
        got = out.cpu().numpy()
        for d in range(4):
            assert_bit_exact(np.ascontiguousarray(got[d, c0:c0 + n]), oracle.xengine(x[d * 48:(d + 1) * 48].numpy(), chans=list(range(c0, c0 + n))))
        assert (got[:, :c0] == 77).all() and (got[:, c0 + n:] == 77).all()
        oh = torch.full(h.output_shape(), 99, dtype=torch.int32)
        h.xengine_host(x, None)
        h.xengine_host(x, oh, accumulate=True)
        assert_bit_exact(np.ascontiguousarray(oh.numpy()[c0:c0 + n]), 2 * want[c0:c0 + n])
        assert (oh[:c0] == 99).all() and (oh[c0 + n:] == 99).all()


def test_window_argument_errors(corr):
    L = corr.lib()
    assert not L.corr_create_window(8, 2, 4, 3, 2, 16, 0)            # window runs past the band
    assert b"window" in L.corr_last_error(None)
    assert not L.corr_create_window(8, 2, 4, -1, 2, 16, 0)
    assert not L.corr_create_window(8, 2, 4, 0, 0, 16, 0)
    with corr.Correlator(8, 2, 4, 16, "ci8", window=(1, 2)) as h:
        x = torch.zeros(h.input_shape(), dtype=torch.int8, device="cuda")
        ws = torch.empty(max(h.workspace_bytes, 128), dtype=torch.uint8, device="cuda")
        assert L.corr_corner_turn(h._h, x.data_ptr(), ws.data_ptr(), None) == corr.CORR_EINVAL


@pytest.mark.parametrize("N,P,C,T,dtype", [(40, 2, 19, 300, "ci8"), (16, 2, 3, 64, "ci8"), (24, 2, 1, 100, "ci8"), (20, 2, 9, 260, "cf16")])
def test_host_path_pipeline(corr, oracle, N, P, C, T, dtype):
    """corr_xengine_host: the channel-window copy pipeline (8 windows, fewer when C < 8) from PINNED and from pageable
    host memory, three calls (store, accumulate, accumulate with readback)."""
    xs = [(inputs.gauss_ci8(T, C, N, P, 40.0, seed=7960 + k) if dtype == "ci8" else inputs.corr_phase_cf16(T, C, N, P, seed=7960 + k))
          for k in range(3)]
    want = run_oracle(oracle, xs)
    for pinned in (True, False):
        with corr.Correlator(N, P, C, T, dtype) as h:
            oh = torch.empty(h.output_shape(), dtype=torch.int32 if dtype == "ci8" else torch.float32)
            if pinned:
                oh = oh.pin_memory()
            for k, x in enumerate(xs):
                xh = x.pin_memory() if pinned else x
                h.xengine_host(xh, oh if k == 2 else None, accumulate=k > 0)
            assert h.last_launch_count == min(C, 8)
            if dtype == "ci8":
                assert_bit_exact(oh.numpy(), want)
            else:
                assert fp16_normalised_error(oh.numpy(), want, N, P) <= FP16_TOL


def test_host_path_accumulate_needs_a_complete_integration(corr):
    """corr_xengine_host keeps its running sum on the device: accumulate != 0 is refused until a call with
    accumulate == 0 has gone through on this handle (the same flag is cleared when a call fails part-way)."""
    x = inputs.gauss_ci8(64, 3, 16, 2, 30.0, seed=7990)
    with corr.Correlator(16, 2, 3, 64, "ci8") as h:
        oh = torch.empty(h.output_shape(), dtype=torch.int32)
        with pytest.raises(corr.CorrError) as ei:
            h.xengine_host(x, oh, accumulate=True)
        assert ei.value.code == corr.CORR_EINVAL and "accumulate without" in str(ei.value)
        h.xengine_host(x, oh)
        h.xengine_host(x, oh, accumulate=True)
        first = oh.clone()
        h.xengine_host(x, oh)
        assert torch.equal(2 * oh, first)


# ---------------------------------------------------------------------------------------------
# rectangular cross-only X-engine (corr_xengine_cross) against oracle.xengine_cross
# ---------------------------------------------------------------------------------------------
def run_cross(corr, xa, xb, dtype, calls=1, kernel=None):
    T, C, Na, P, _ = xa.shape
    Nb = xb.shape[2]
    with corr.CrossCorrelator(Na, Nb, P, C, T, dtype) as h:
        if kernel is not None:
            h.set_kernel(kernel)
            assert h.kernel == kernel
        out = None
        for k in range(calls):
            out = h.xengine_cross(xa.cuda(), xb.cuda(), out, accumulate=k > 0)
        torch.cuda.synchronize()
        return out.cpu().numpy(), h.kernel


CROSS_CASES = [(1, 1, 1, 1, 1), (4, 4, 2, 3, 70), (16, 48, 2, 5, 130), (64, 64, 2, 4, 200), (72, 136, 2, 2, 129),
               (200, 60, 2, 2, 64), (130, 70, 1, 3, 96), (33, 8, 2, 2, 50), (128, 256, 2, 2, 257)]


@pytest.mark.parametrize("kernel", [None, "simt"])
@pytest.mark.parametrize("Na,Nb,P,C,T", CROSS_CASES)
def test_cross_ci8_bit_exact(corr, oracle, kernel, Na, Nb, P, C, T):
    xa = inputs.gauss_ci8(T, C, Na, P, 40.0, seed=7300 + Na)
    xb = inputs.gauss_ci8(T, C, Nb, P, 40.0, seed=7400 + Nb)
    got, used = run_cross(corr, xa, xb, "ci8", calls=2, kernel=kernel)
    tma = (Na * P * 2) % 16 == 0 and (Nb * P * 2) % 16 == 0
    assert used == ("pair" if tma and kernel is None else "simt")
    want = oracle.xengine_cross(xa.numpy(), xb.numpy())
    want = oracle.xengine_cross(xa.numpy(), xb.numpy(), accumulate_into=want)
    assert got.dtype == np.int32 and got.shape == want.shape
    bad = np.argwhere(got.astype(np.int64) != want)
    assert bad.size == 0, "first mismatches (c,i,j,p,q,reim): %s" % bad[:8].tolist()


@pytest.mark.parametrize("Na,Nb,P,C,T", [(24, 40, 2, 3, 100), (64, 160, 2, 2, 2100), (96, 32, 1, 2, 1030)])
def test_cross_cf16_within_tolerance(corr, oracle, Na, Nb, P, C, T):
    x = inputs.corr_phase_cf16(T, C, Na + Nb, P, seed=7500 + Na)      # one sky, two station groups
    xa, xb = x[:, :, :Na].contiguous(), x[:, :, Na:].contiguous()
    got, used = run_cross(corr, xa, xb, "cf16")
    assert used == "pair"
    want = oracle.xengine_cross(xa.numpy(), xb.numpy())
    # |dV_ij| <= 2e-5 sqrt(V_ii V_jj): autocorrelations of each group from the (pinned) triangle oracle
    auto_a = oracle.xengine(xa.numpy())[:, [i * (i + 1) // 2 + i for i in range(Na)]]
    auto_b = oracle.xengine(xb.numpy())[:, [j * (j + 1) // 2 + j for j in range(Nb)]]
    pa = np.stack([auto_a[:, :, p, p, 0] for p in range(P)], axis=-1)           # [C, Na, P]
    pb = np.stack([auto_b[:, :, q, q, 0] for q in range(P)], axis=-1)           # [C, Nb, P]
    d = got.astype(np.float64) - want
    err = np.sqrt(d[..., 0] ** 2 + d[..., 1] ** 2) / np.sqrt(pa[:, :, None, :, None] * pb[:, None, :, None, :])
    assert err.max() <= FP16_TOL, "normalised error %.3g" % err.max()


def test_cross_matches_the_triangle_kernel_block(corr):
    """GPU against GPU: the rectangle of stations [k, N) x [0, k) equals the triangle kernel's off-diagonal block."""
    T, C, N, P, k = 256, 3, 96, 2, 40
    x = inputs.gauss_ci8(T, C, N, P, 30.0, seed=7600)
    tri, _ = run_gpu(corr, [x], "ci8")
    got, _ = run_cross(corr, x[:, :, k:].contiguous(), x[:, :, :k].contiguous(), "ci8")
    for i in range(k, N):
        assert (got[:, i - k] == tri[:, i * (i + 1) // 2: i * (i + 1) // 2 + k]).all()


def test_cross_argument_errors(corr):
    with corr.CrossCorrelator(8, 16, 2, 2, 64, "ci8") as h, corr.Correlator(8, 2, 2, 64, "ci8") as g:
        L = corr.lib()
        xa = torch.zeros(h.input_shape(), dtype=torch.int8, device="cuda")
        xb = torch.zeros(h.input_shape_b(), dtype=torch.int8, device="cuda")
        out = h.empty_output()
        assert h.input_bytes == xa.numel() and h.input_bytes_b == xb.numel() and h.output_bytes == out.numel() * 4
        assert L.corr_xengine(h._h, xa.data_ptr(), out.data_ptr(), 0, None) == corr.CORR_EINVAL        # wrong entry point
        assert L.corr_xengine_cross(g._h, xa.data_ptr(), xb.data_ptr(), out.data_ptr(), 0, None) == corr.CORR_EINVAL
        assert L.corr_xengine_cross(h._h, xa.data_ptr(), None, out.data_ptr(), 0, None) == corr.CORR_EINVAL
        assert L.corr_xengine_cross(h._h, xa.data_ptr(), xb.data_ptr() + 2, out.data_ptr(), 0, None) == corr.CORR_EINVAL
        with pytest.raises(corr.CorrError):
            h.set_kernel("single")
    assert not corr.lib().corr_create_cross(4, 0, 2, 1, 1, 0)


# ---------------------------------------------------------------------------------------------
# short-integration mode (corr_xengine_dumps): every dump is Eq. 2 on its own slice of samples
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("N,P,C,T,n_dump", [(16, 2, 5, 300, 3), (64, 2, 4, 512, 4), (72, 2, 3, 260, 2), (136, 1, 2, 384, 3),
                                            (256, 2, 2, 256, 8), (33, 2, 2, 90, 3), (80, 2, 3, 64, 64)])
def test_dumps_ci8_bit_exact(corr, oracle, N, P, C, T, n_dump):
    x = inputs.gauss_ci8(T, C, N, P, 40.0, seed=7700 + N + n_dump)
    with corr.Correlator(N, P, C, T, "ci8") as h:
        got = h.xengine_dumps(x.cuda(), n_dump).cpu().numpy()
        whole = h.xengine(x.cuda()).cpu().numpy()                 # the same handle still integrates the whole block
    Ts = T // n_dump
    assert got.shape[0] == n_dump
    for d in range(n_dump):
        assert_bit_exact(got[d], oracle.xengine(x[d * Ts:(d + 1) * Ts].numpy()))
    assert (got.astype(np.int64).sum(axis=0) == whole).all()      # additivity in time (pin 8) through the GPU path
    assert_bit_exact(whole, oracle.xengine(x.numpy()))


def test_dumps_cf16_within_tolerance(corr, oracle):
    N, P, C, T, n_dump = 48, 2, 3, 2400, 2                       # 1200 samples per dump: two TMEM passes each
    x = inputs.corr_phase_cf16(T, C, N, P, seed=7800)
    with corr.Correlator(N, P, C, T, "cf16") as h:
        got = h.xengine_dumps(x.cuda(), n_dump).cpu().numpy()
    for d in range(n_dump):
        want = oracle.xengine(x[d * 1200:(d + 1) * 1200].numpy())
        assert fp16_normalised_error(got[d], want, N, P) <= FP16_TOL


def test_dumps_argument_errors(corr):
    with corr.Correlator(16, 2, 2, 96, "ci8") as h, corr.CrossCorrelator(8, 8, 2, 2, 64, "ci8") as g:
        L = corr.lib()
        x = torch.zeros(h.input_shape(), dtype=torch.int8, device="cuda")
        out = torch.empty((4,) + tuple(h.output_shape()), dtype=torch.int32, device="cuda")
        assert L.corr_xengine_dumps(h._h, x.data_ptr(), out.data_ptr(), 5, None) == corr.CORR_EINVAL     # 5 does not divide 96
        assert L.corr_xengine_dumps(h._h, x.data_ptr(), out.data_ptr(), 0, None) == corr.CORR_EINVAL
        assert L.corr_xengine_dumps(h._h, None, out.data_ptr(), 4, None) == corr.CORR_EINVAL
        assert L.corr_xengine_dumps(g._h, x.data_ptr(), out.data_ptr(), 4, None) == corr.CORR_EINVAL     # cross plan
        assert L.corr_xengine_dumps(None, x.data_ptr(), out.data_ptr(), 4, None) == corr.CORR_EINVAL


@pytest.mark.parametrize("kernel,N,P,C,T", [("single", 16, 2, 64, 256), ("pair", 136, 2, 21, 260)])
def test_cuda_graph_capture_of_an_accumulate_sequence(corr, oracle, kernel, N, P, C, T):
    """corr.h: a sequence of corr_xengine calls (store, accumulate, accumulate) captured with stream capture and replayed
    reproduces the oracle's integration bit for bit on every replay (the tile-feed counter memset is part of the graph)."""
    xs = [inputs.gauss_ci8(T, C, N, P, 30.0, seed=9900 + k).cuda() for k in range(3)]
    want = None
    for x in xs:
        want = oracle.xengine(x.cpu().numpy(), accumulate_into=want)
    with corr.Correlator(N, P, C, T, "ci8") as h:
        h.set_kernel(kernel)
        out = h.empty_output()
        for k, x in enumerate(xs):                                   # once outside the capture
            h.xengine(x, out, accumulate=k > 0)
        torch.cuda.synchronize()
        s = torch.cuda.Stream()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.stream(s):
            with torch.cuda.graph(g, stream=s):
                for k, x in enumerate(xs):
                    h.xengine(x, out, accumulate=k > 0, stream=s)
        for rep in range(3):
            out.fill_(-7)                                            # every replay starts from garbage and must overwrite it
            g.replay()
            torch.cuda.synchronize()
            assert (out.cpu().numpy().astype(np.int64) == want).all()
