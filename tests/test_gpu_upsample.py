"""GPU parity of lisa_td_link_response_up2 (reading A20): polarisations computed
on the 2 dt grid, linearly interpolated to the dt grid while the strain tile is staged."""
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


@pytest.mark.parametrize("order", [1, 31])
def test_link_response_up2_parity(lib, orc, order):
    B, N = 3, 1 << 13
    fine = synth.make_inputs(3, B=B, N=N + 2)      # N/2 + 1 coarse samples = every other fine one
    Nc = N // 2 + 1
    co = lambda k: fine[k][..., ::2].contiguous()
    amp, phase, al, be, ga = co("amp"), co("phase"), co("alpha"), co("beta"), co("gamma")
    assert amp.shape[-1] == Nc
    n = lambda t: t.numpy()
    dt, t0 = fine["dt"], fine["t0"]
    hp_ref, hc_ref = orc.modes_to_pol(fine["l"], fine["m"], n(amp), n(phase), n(fine["iota"]), n(fine["phi"]),
                                      n(fine["psi"]), n(al), n(be), n(ga))
    y_ref = orc.link_response(orc.upsample2(hp_ref), orc.upsample2(hc_ref), n(fine["lam"]), n(fine["beta_sky"]),
                              fine["orbit"], t0, dt, order, fine["margin_y"])
    hp = torch.empty((B, Nc), dtype=torch.float64, device="cuda")
    hc = torch.empty_like(hp)
    lib.modes_to_pol(B, Nc, fine["l"], fine["m"], amp.cuda(), phase.cuda(), al.cuda(), be.cuda(), ga.cuda(),
                     fine["iota"].cuda(), fine["phi"].cuda(), fine["psi"].cuda(), None, hp, hc)
    y = torch.full((B, 6, N), float("nan"), dtype=torch.float64, device="cuda")
    lib.link_response_up2(B, N, t0, dt, order, fine["margin_y"], hp, hc, fine["lam"].cuda(), fine["beta_sky"].cuda(),
                          fine["orbit"], y)
    torch.cuda.synchronize()
    got = y.cpu().numpy()
    m = fine["margin_y"]
    assert np.all(got[:, :, :m] == 0) and np.all(got[:, :, N - m:] == 0)
    for b in range(B):
        for l in range(6):
            err = np.linalg.norm(got[b, l] - y_ref[b, l]) / np.linalg.norm(y_ref[b, l])
            assert err < 2e-13, (b, l, err)


def test_up2_rejects_odd_length(lib):
    z = torch.zeros(4096, dtype=torch.float64, device="cuda")
    with pytest.raises(lib.LisaTdError):
        lib.link_response_up2(1, 4097, 0.0, 5.0, 31, 128, z, z, z[:1], z[:1], synth.kepler_orbit(), z)


def test_pipeline_host_up2_matches_the_oracle(lib, orc):
    """the end-to-end call with modes on the 2 dt grid: chunks of 2 walkers over B = 5,
    against oracle S1 on the coarse grid -> linear upsampling -> S2, S3, S4/S5"""
    B, N = 5, 1 << 13
    fine = synth.make_inputs(4, B=B, N=N + 2)
    Nc = N // 2 + 1
    co = lambda k: fine[k][..., ::2].contiguous()
    amp, phase, al, be, ga = co("amp"), co("phase"), co("alpha"), co("beta"), co("gamma")
    n = lambda t: t.numpy()
    dt, t0, order = fine["dt"], fine["t0"], fine["order"]
    hp_c, hc_c = orc.modes_to_pol(fine["l"], fine["m"], n(amp), n(phase), n(fine["iota"]), n(fine["phi"]),
                                  n(fine["psi"]), n(al), n(be), n(ga))
    y_ref = orc.link_response(orc.upsample2(hp_c), orc.upsample2(hc_c), n(fine["lam"]), n(fine["beta_sky"]),
                              fine["orbit"], t0, dt, order, fine["margin_y"])
    tdi_ref = orc.tdi(y_ref, fine["orbit"], t0, dt, order, 20, 1, fine["margin_lo"], fine["margin_hi"])
    kmin, kmax = synth.likelihood_band(N, dt)
    w = orc.psd_weights(N, dt, synth.NOISE["acc"], synth.NOISE["oms"], synth.NOISE["arm_s"], 20)
    data = orc.spectrum3(tdi_ref[0])
    ref_ll, ref_dh, ref_hh = orc.loglike(tdi_ref, data, w, kmin, kmax)
    pipe = lib.Pipeline(2, N, len(fine["l"]), True)
    pin = lambda t: t.contiguous().pin_memory()
    out = [torch.empty(B, dtype=torch.float64).pin_memory() for _ in range(3)]
    lib.pipeline_host_up2(pipe, B, N, fine["l"], fine["m"], pin(amp), pin(phase), pin(al), pin(be), pin(ga),
                          pin(fine["iota"]), pin(fine["phi"]), pin(fine["psi"]), pin(fine["lam"]), pin(fine["beta_sky"]),
                          t0, dt, order, fine["margin_y"], 20, fine["margin_lo"], fine["margin_hi"], fine["orbit"],
                          pin(torch.from_numpy(data)), pin(torch.from_numpy(w)), kmin, kmax, out[0], out[1], out[2])
    for got, ref in zip(out, (ref_ll, ref_dh, ref_hh)):
        err = np.max(np.abs(got.numpy() - ref) / np.abs(ref))
        assert err < 1e-9, err
    pipe.close()
