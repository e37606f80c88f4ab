"""GPU parity of lisa_td_fisher (reading A19) against the long-double oracle.

Stage parity feeds both sides the SAME A,E,T series, so only the FFT and the reduction differ
(bar 1e-11 of sqrt(G_ii G_jj)).  The chain test runs D+1 perturbed walkers through S1..S3 on
each side: a forward difference with a relative step s amplifies the ~5e-13 error of the TDI
series by 1/s, so with s = 1e-3 the bar is 1e-8 of sqrt(G_ii G_jj).
"""
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


def _gpu_fisher(lib, tdi, delta, w, kmin, kmax):
    D, N = tdi.shape[0] - 1, tdi.shape[-1]
    plan = lib.Plan(D + 1, N)
    out = torch.full((D, D), float("nan"), dtype=torch.float64, device="cuda")
    lib.fisher(plan, D, N, torch.from_numpy(np.ascontiguousarray(tdi)).cuda(), delta, torch.from_numpy(w).cuda(),
               kmin, kmax, out)
    torch.cuda.synchronize()
    plan.close()
    return out.cpu().numpy()


def _rel(got, ref):
    s = np.sqrt(np.abs(np.diag(ref)))
    return np.max(np.abs(got - ref) / np.outer(s, s))


@pytest.mark.parametrize("D,N,band", [(1, 4096, (5, 400)), (7, 4096, (0, 2048)), (32, 2048, (17, 901)), (15, 1 << 14, (33, 6553))])
def test_fisher_stage_parity(lib, orc, D, N, band):
    rng = np.random.default_rng(D + N)
    tdi = rng.standard_normal((D + 1, 3, N))
    delta = rng.uniform(0.1, 2.0, D) * rng.choice([-1.0, 1.0], D)
    w = rng.uniform(0.5, 2.0, (3, N // 2 + 1))
    ref = orc.fisher(tdi, delta, w, *band)
    got = _gpu_fisher(lib, tdi, delta, w, *band)
    assert np.all(got == got.T)
    assert _rel(got, ref) < 1e-11


def test_fisher_rejects_bad_arguments(lib):
    N = 2048
    plan = lib.Plan(4, N)
    z = torch.zeros((5, 3, N), dtype=torch.float64, device="cuda")
    w = torch.ones((3, N // 2 + 1), dtype=torch.float64, device="cuda")
    out = torch.zeros((4, 4), dtype=torch.float64, device="cuda")
    with pytest.raises(lib.LisaTdError):   # D + 1 walkers exceed the plan
        lib.fisher(plan, 4, N, z, np.ones(4), w, 1, 100, out)
    with pytest.raises(lib.LisaTdError):   # zero step
        lib.fisher(plan, 3, N, z, np.array([1.0, 0.0, 1.0]), w, 1, 100, out)
    plan.close()


def test_fisher_chain_extrinsic_parameters(lib, orc):
    """Five extrinsic parameters (iota, phi, psi, lambda, beta_sky) of a configs[3]-shaped
    walker, perturbed by 1e-3 rad each, through S1..S3 on both sides."""
    N, rel_step = 1 << 14, 1e-3
    names = ["iota", "phi", "psi", "lam", "beta_sky"]
    D = len(names)
    inp = synth.make_inputs(4, B=1, N=N)
    inp = {k: (v.repeat((D + 1,) + (1,) * (v.dim() - 1)).contiguous() if isinstance(v, torch.Tensor) else v)
           for k, v in inp.items()}
    delta = np.full(D, rel_step)
    for i, nm in enumerate(names):
        inp[nm][i + 1] += delta[i]
    B = D + 1
    dt = inp["dt"]
    kmin, kmax = synth.likelihood_band(N, dt)
    w = orc.psd_weights(N, dt, synth.NOISE["acc"], synth.NOISE["oms"], synth.NOISE["arm_s"], 20)
    n = lambda k: None if inp[k] is None else inp[k].numpy()
    ref_tdi = orc.chain(inp["l"], inp["m"], n("amp"), n("phase"), n("iota"), n("phi"), n("psi"), n("lam"),
                        n("beta_sky"), inp["orbit"], inp["t0"], dt, inp["order"], inp["margin_y"], 20, 1,
                        inp["margin_lo"], inp["margin_hi"], alpha=n("alpha"), beta=n("beta"), gamma=n("gamma"),
                        want=("tdi",))["tdi"]
    ref = orc.fisher(ref_tdi, delta, w, kmin, kmax)
    d = lambda k: None if inp[k] is None else inp[k].cuda()
    hp = torch.empty((B, N), dtype=torch.float64, device="cuda")
    hc = torch.empty_like(hp)
    y = torch.empty((B, 6, N), dtype=torch.float64, device="cuda")
    tdi = torch.empty((B, 3, N), dtype=torch.float64, device="cuda")
    lib.modes_to_pol(B, N, inp["l"], inp["m"], d("amp"), d("phase"), d("alpha"), d("beta"), d("gamma"),
                     d("iota"), d("phi"), d("psi"), None, hp, hc)
    lib.link_response(B, N, inp["t0"], dt, inp["order"], inp["margin_y"], hp, hc, d("lam"), d("beta_sky"),
                      inp["orbit"], y)
    lib.tdi2(B, N, inp["t0"], dt, inp["order"], 20, 1, inp["margin_lo"], inp["margin_hi"], y, inp["orbit"], tdi)
    plan = lib.Plan(B, N)
    out = torch.empty((D, D), dtype=torch.float64, device="cuda")
    lib.fisher(plan, D, N, tdi, delta, torch.from_numpy(w).cuda(), kmin, kmax, out)
    torch.cuda.synchronize()
    plan.close()
    got = out.cpu().numpy()
    err = _rel(got, ref)
    print("Fisher chain error:", err, "diag", np.diag(ref))
    assert err < 1e-8
    assert np.all(np.linalg.eigvalsh(got) > 0)
