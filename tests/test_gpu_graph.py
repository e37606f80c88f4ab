"""The C-ABI calls only enqueue work on the caller's stream, so a whole S1..S5 evaluation can be captured
into a CUDA graph and replayed (launch-bound small problems: configs[0] is 5 kernels + 2 cuFFT kernels
of a few microseconds each)."""
import numpy as np
import pytest
import torch

from paper_2501_08261_b200 import synth

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def lib():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2501_08261_b200 import lib as L
    L.load()
    return L


@pytest.mark.parametrize("config,B,N", [(1, 1, 1 << 12), (3, 4, 1 << 14)])
def test_chain_replays_from_a_cuda_graph(lib, config, B, N):
    inp = synth.make_inputs(config, device="cuda", B=B, N=N)
    dt, t0 = inp["dt"], inp["t0"]
    f64 = torch.float64
    hp = torch.empty((B, N), dtype=f64, device="cuda")
    hc = torch.empty_like(hp)
    y = torch.empty((B, 6, N), dtype=f64, device="cuda")
    tdi = torch.empty((B, 3, N), dtype=f64, device="cuda")
    ll = torch.empty(B, dtype=f64, device="cuda")
    nf = N // 2 + 1
    data = torch.randn((3, nf, 2), dtype=f64, device="cuda") * 1e-18
    w = torch.from_numpy(lib.psd_weights(N, dt, synth.NOISE["acc"], synth.NOISE["oms"], synth.NOISE["arm_s"], 20)).cuda()
    kmin, kmax = synth.likelihood_band(N, dt)
    plan = lib.Plan(B, N)
    g = lambda k: inp[k]

    def chain():
        lib.modes_to_pol(B, N, inp["l"], inp["m"], g("amp"), g("phase"), g("alpha"), g("beta"), g("gamma"), g("iota"),
                         g("phi"), g("psi"), None, hp, hc)
        lib.link_response(B, N, t0, dt, inp["order"], inp["margin_y"], hp, hc, g("lam"), g("beta_sky"), inp["orbit"], y)
        lib.tdi2(B, N, t0, dt, inp["order"], 20, 1, inp["margin_lo"], inp["margin_hi"], y, inp["orbit"], tdi)
        lib.loglike(plan, B, N, tdi, data, w, kmin, kmax, ll)

    chain()  # eager: also creates the cuFFT plan of this batch size
    torch.cuda.synchronize()
    want_ll, want_tdi = ll.clone(), tdi.clone()
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.stream(side):
        chain()  # warm-up on the capture stream
        with torch.cuda.graph(graph, stream=side):
            chain()
    torch.cuda.current_stream().wait_stream(side)
    ll.zero_()
    tdi.zero_()
    # new inputs in the same buffers: the graph must recompute from them
    inp["phase"].add_(0.25)
    chain()
    torch.cuda.synchronize()
    moved_ll = ll.clone()
    assert not torch.equal(moved_ll, want_ll)
    ll.zero_()
    graph.replay()
    torch.cuda.synchronize()
    assert torch.equal(ll, moved_ll)          # same kernels, same bits
    inp["phase"].sub_(0.25)
    graph.replay()
    torch.cuda.synchronize()
    assert torch.allclose(ll, want_ll, rtol=1e-12, atol=0.0)
    assert torch.allclose(tdi, want_tdi, rtol=0.0, atol=1e-12 * float(want_tdi.abs().max()))
    # replay rate against eager launches
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
    ev[0].record()
    for _ in range(50):
        chain()
    ev[1].record()
    for _ in range(50):
        graph.replay()
    ev[2].record()
    torch.cuda.synchronize()
    print(f"config {config} B={B} N={N}: eager {ev[0].elapsed_time(ev[1]) / 50 * 1e3:.1f} us, graph replay "
          f"{ev[1].elapsed_time(ev[2]) / 50 * 1e3:.1f} us per evaluation")
    plan.close()
