"""Race / lifetime stress of the tensor-core kernels (compute-sanitizer is closed on the GPU pool, profiles/r2_sanitizer.md):
what a data race in the barrier pipeline, the cross-CTA tile feed, the TMEM hand-over or the staging-buffer reuse would
produce is a wrong or a run-to-run DIFFERENT output, so these tests launch the same work hundreds of times -- back to
back, on two streams at once, with inputs and accumulate flags alternating -- and demand bit-identical, oracle-exact
results every time.  The writer additionally bounds-checks every bulk store in the kernel (a violation traps)."""
import numpy as np
import pytest
import torch

from paper_1305_5639_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def corr():
    from paper_1305_5639_b200 import binding
    binding.lib()
    return binding


@pytest.mark.parametrize("kernel,N,P,C,T", [("pair", 136, 2, 37, 300), ("pair", 256, 2, 9, 520), ("single", 40, 2, 151, 200),
                                            ("pair", 72, 1, 50, 129)])
def test_repeated_launches_are_bit_identical_ci8(corr, oracle, kernel, N, P, C, T):
    """200 back-to-back launches (more tiles than co-resident clusters, ragged tiles, T not a multiple of the stage):
    every output equals the first, and the first equals the oracle."""
    x = inputs.gauss_ci8(T, C, N, P, 40.0, seed=8100 + N).cuda()
    want = oracle.xengine(x.cpu().numpy())
    with corr.Correlator(N, P, C, T, "ci8") as h:
        h.set_kernel(kernel)
        first = h.xengine(x)
        torch.cuda.synchronize()
        assert (first.cpu().numpy().astype(np.int64) == want).all()
        outs = [h.empty_output() for _ in range(4)]
        for it in range(200):
            h.xengine(x, outs[it % 4])
        torch.cuda.synchronize()
        for o in outs:
            assert torch.equal(o, first)


def test_repeated_launches_are_bit_identical_cf16(corr, oracle):
    """fp16 path, four TMEM passes per tile folded in registers: the summation order is fixed, so repeated launches
    agree bit for bit (and with the oracle within the tolerance)."""
    N, P, C, T = 128, 2, 20, 4100
    x = inputs.corr_phase_cf16(T, C, N, P, seed=8200).cuda()
    with corr.Correlator(N, P, C, T, "cf16") as h:
        first = h.xengine(x)
        outs = [h.empty_output() for _ in range(3)]
        for it in range(60):
            h.xengine(x, outs[it % 3])
        torch.cuda.synchronize()
        for o in outs:
            assert torch.equal(o, first)
    want = oracle.xengine(x.cpu().numpy(), chans=[0, 7, 19])
    got = first.cpu().numpy()[[0, 7, 19]].astype(np.float64)
    auto_b = np.array([i * (i + 1) // 2 + i for i in range(N)])
    i_of_b = np.concatenate([np.full(i + 1, i) for i in range(N)])
    j_of_b = np.concatenate([np.arange(i + 1) for i in range(N)])
    auto = np.stack([want[:, auto_b, p, p, 0] for p in range(P)], axis=-1)
    d = got - want
    err = np.sqrt(d[..., 0] ** 2 + d[..., 1] ** 2) / np.sqrt(auto[:, i_of_b, :, None] * auto[:, j_of_b, None, :])
    assert err.max() <= 2e-5


def test_two_streams_two_handles_concurrently(corr, oracle):
    """Two handles on two streams, launches interleaved from the host so that kernels of both are in flight together
    (each launch takes its own tile-feed counter); accumulate sequences of three different inputs."""
    N, P, C, T = 136, 2, 21, 260
    xs = [inputs.gauss_ci8(T, C, N, P, 40.0, seed=8300 + k).cuda() for k in range(3)]
    want = None
    for x in xs:
        want = oracle.xengine(x.cpu().numpy(), accumulate_into=want)
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    with corr.Correlator(N, P, C, T, "ci8") as h1, corr.Correlator(N, P, C, T, "ci8") as h2:
        h1.set_kernel("pair")
        h2.set_kernel("pair")
        o1, o2 = h1.empty_output(), h2.empty_output()
        torch.cuda.synchronize()
        for rep in range(40):
            for k, x in enumerate(xs):
                h1.xengine(x, o1, accumulate=k > 0, stream=s1)
                h2.xengine(xs[2 - k], o2, accumulate=k > 0, stream=s2)      # the same sum in the opposite order
            if rep % 8 == 7:
                torch.cuda.synchronize()
                assert (o1.cpu().numpy().astype(np.int64) == want).all()
                assert (o2.cpu().numpy().astype(np.int64) == want).all()


def test_cross_and_dumps_repeated(corr, oracle):
    xa = inputs.gauss_ci8(200, 9, 136, 2, 30.0, seed=8400).cuda()
    xb = inputs.gauss_ci8(200, 9, 72, 2, 30.0, seed=8401).cuda()
    want = oracle.xengine_cross(xa.cpu().numpy(), xb.cpu().numpy())
    with corr.CrossCorrelator(136, 72, 2, 9, 200, "ci8") as h:
        outs = [h.empty_output() for _ in range(3)]
        for it in range(90):
            h.xengine_cross(xa, xb, outs[it % 3])
        torch.cuda.synchronize()
        for o in outs:
            assert (o.cpu().numpy().astype(np.int64) == want).all()
    x = inputs.gauss_ci8(256, 11, 136, 2, 30.0, seed=8402).cuda()
    with corr.Correlator(136, 2, 11, 256, "ci8") as h:
        first = h.xengine_dumps(x, 8)
        for d in range(8):
            assert (first[d].cpu().numpy().astype(np.int64) == oracle.xengine(x[d * 32:(d + 1) * 32].cpu().numpy())).all()
        for it in range(400):                                 # 1-stage tiles: the fastest tile turnover the feed sees
            assert torch.equal(h.xengine_dumps(x, 8), first)


def test_fengine_tensor_core_long_queues_under_dram_load(corr):
    """The tensor-core F-engine with hundreds of tiles per CTA, input and output far larger than L2, launched repeatedly:
    TMA loads then complete out of order and the hand-overs of the raw ring, the A buffers in tensor memory and the two
    accumulators see every interleaving.  (Round 2: waiting on a ring slot before the A buffer let a fast fold warp meet
    the slot's barrier one phase behind -- 1 launch in 15 of this geometry failed, none of the small parity cases.)
    Every launch must reproduce the first bit for bit, and the first must agree with the CUDA-core kernel."""
    M, A = 512, 4096
    g = torch.Generator(device="cuda")
    g.manual_seed(8500)
    s = torch.clamp(torch.round(torch.randn((M, A * 256), generator=g, device="cuda") * 20.0), -127, 127).to(torch.int8)
    assert corr.fengine_uses_tensor_cores(M)
    first = corr.fengine(s)
    torch.cuda.synchronize()
    ref = corr.fengine(s, simt=True)
    # the two kernels round the same exact value through different fp32 sums: one fp16 ulp of the largest magnitude apart
    d = (first.float() - ref.float()).abs().max().item()
    assert d <= 2.0 * float(torch.finfo(torch.float16).eps) * ref.float().abs().max().item() + 1e-3
    del ref
    out = torch.empty_like(first)
    for it in range(120):
        corr.fengine(s, out)
        if it % 20 == 19:
            torch.cuda.synchronize()
            assert torch.equal(out, first)


def test_fengine_ci8_tensor_core_long_queues(corr):
    """The requantised int8 variant of the tensor-core F-engine (4-deep raw ring, pair exchange buffers and named
    barriers in the epilogue) under the same load: repeated launches are bit-identical, and the codes agree with the
    CUDA-core kernel's except within one code at rounding ties of the two kernels' fp32 sums (< 1 % of the components)."""
    M, A = 512, 2048
    g = torch.Generator(device="cuda")
    g.manual_seed(8600)
    s = torch.clamp(torch.round(torch.randn((M, A * 256), generator=g, device="cuda") * 20.0), -127, 127).to(torch.int8)
    first = corr.fengine(s, scale=1.0 / 20)
    torch.cuda.synchronize()
    # CUDA-core reference on a stream count that is not a multiple of 64 (the first 500 streams)
    ref = corr.fengine(s[:500].contiguous(), scale=1.0 / 20)
    d = (first[:, :, :500].to(torch.int16) - ref.to(torch.int16)).abs()
    assert d.max().item() <= 1 and (d != 0).float().mean().item() < 1e-2
    del ref, d
    out = torch.empty_like(first)
    for it in range(120):
        corr.fengine(s, out, scale=1.0 / 20)
        if it % 20 == 19:
            torch.cuda.synchronize()
            assert torch.equal(out, first)
