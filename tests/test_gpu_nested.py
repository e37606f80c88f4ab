"""GPU parity of the delay model of reading A22: first-order light travel times
(`tt_order` 1) in S2, S3 and the laser helper, and TDI delays chained along the light path
(`nested` 1) in S3 -- merged-stencil DMMA kernel and generic kernel, KEPLER1 and TABLE orbits."""
import numpy as np
import pytest
import torch

from paper_2501_08261_b200 import synth

pytestmark = pytest.mark.gpu
S = [3, 1, 2, 2, 3, 1]
R = [2, 3, 1, 3, 1, 2]


@pytest.fixture(scope="module")
def lib():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2501_08261_b200 import lib as L
    L.load()
    return L


def _table_orbit(orc, t_lo, t_hi, order=7, h=86400.0):
    kep = synth.kepler_orbit()
    n_tab = int(np.ceil((t_hi - t_lo) / h)) + 1 + order
    t0 = t_lo - (order // 2) * h
    tab = np.stack([orc.orbit_eval(kep, t0 + h * j)[0] for j in range(n_tab)])
    return {"kind": "table", "r_tab": tab, "t_tab0": t0, "dt_tab": h, "tab_order": order}


def _chain_both(lib, orc, inp, orbit, B, N, t0, generation, out_kind):
    dt = inp["dt"]
    n = lambda k: None if inp[k] is None else inp[k].numpy()
    ref = orc.chain(inp["l"], inp["m"], n("amp"), n("phase"), n("iota"), n("phi"), n("psi"), n("lam"), n("beta_sky"),
                    orbit, t0, dt, inp["order"], inp["margin_y"], generation, out_kind, inp["margin_lo"],
                    inp["margin_hi"], alpha=n("alpha"), beta=n("beta"), gamma=n("gamma"), want=("y", "tdi"))
    d = lambda k: None if inp[k] is None else inp[k].cuda()
    hp = torch.empty((B, N), dtype=torch.float64, device="cuda")
    hc = torch.empty_like(hp)
    y = torch.empty((B, 6, N), dtype=torch.float64, device="cuda")
    tdi = torch.empty((B, 3, N), dtype=torch.float64, device="cuda")
    lib.modes_to_pol(B, N, inp["l"], inp["m"], d("amp"), d("phase"), d("alpha"), d("beta"), d("gamma"), d("iota"),
                     d("phi"), d("psi"), None, hp, hc)
    lib.link_response(B, N, t0, dt, inp["order"], inp["margin_y"], hp, hc, d("lam"), d("beta_sky"), orbit, y)
    lib.tdi2(B, N, t0, dt, inp["order"], generation, out_kind, inp["margin_lo"], inp["margin_hi"], y, orbit, tdi)
    torch.cuda.synchronize()
    return ref, y.cpu().numpy(), tdi.cpu().numpy()


@pytest.mark.parametrize("kind,generation,out_kind,force_generic", [
    ("kepler1", 20, 1, False), ("kepler1", 15, 0, False), ("table", 20, 1, False), ("kepler1", 20, 0, True)])
def test_chain_with_first_order_travel_times_and_chained_delays(lib, orc, kind, generation, out_kind, force_generic):
    B, N, t0 = 3, 1 << 13, 1.7e6
    inp = synth.make_inputs(3, B=B, N=N)
    base = synth.kepler_orbit() if kind == "kepler1" else _table_orbit(orc, t0, t0 + N * inp["dt"])
    orbit = dict(base, tt_order=1, nested=1)
    lib.debug_force_generic(force_generic)
    try:
        ref, yg, tg = _chain_both(lib, orc, inp, orbit, B, N, t0, generation, out_kind)
    finally:
        lib.debug_force_generic(False)
    for b in range(B):
        for l in range(6):
            err = np.linalg.norm(yg[b, l] - ref["y"][b, l]) / np.linalg.norm(ref["y"][b, l])
            assert err < 5e-13, (b, l, err)
        common = max(np.linalg.norm(ref["tdi"][b, c]) for c in range(3))
        errs = [np.linalg.norm(tg[b, c] - ref["tdi"][b, c]) / common for c in range(3)]
        print(kind, generation, "walker", b, errs)
        assert max(errs) < 1e-11
        lo, hi = inp["margin_lo"], N - inp["margin_hi"]
        assert np.all(tg[b, :, :lo] == 0.0) and np.all(tg[b, :, hi:] == 0.0)
    # the delay model is visible at the bar: the A8/A10 model differs from A22 by far more than 1e-11
    # wherever the TDI output is a small remnant of the links
    ref0, _, _ = _chain_both(lib, orc, inp, dict(base), B, N, t0, generation, out_kind)
    common = max(np.linalg.norm(ref["tdi"][0, c]) for c in range(3))
    assert max(np.linalg.norm(ref0["tdi"][0, c] - ref["tdi"][0, c]) for c in range(3)) / common > 1e-8


def _three_laser_links(orc, orbit, t0, dt, N):
    f = np.array([3.1e-3, 4.7e-3, 6.3e-3], dtype=np.longdouble)
    ph = np.array([0.3, 1.1, 2.5], dtype=np.longdouble)
    t = np.longdouble(t0) + np.arange(N, dtype=np.longdouble) * np.longdouble(dt)
    L = np.array([orc.orbit_eval(orbit, float(tt))[1] for tt in t]).astype(np.longdouble)
    p = lambda i, tt: np.sin(2 * np.pi * f[i] * tt + ph[i])
    y = np.zeros((1, 6, N))
    for l in range(6):
        y[0, l] = (p(S[l] - 1, t - L[:, l]) - p(R[l] - 1, t)).astype(np.float64)
    return y


@pytest.mark.parametrize("order", [31, 7])
def test_three_laser_cancellation_on_the_gpu(lib, orc, order):
    """chained generation 2 on flexing arms with L_l != L_-l cancels three independent lasers to the
    interpolation floor; summed delays leave 1e-8 (order 31: DMMA kernel, order 7: generic kernel)"""
    orbit = dict(synth.kepler_orbit(), tt_order=1)
    N, dt, t0, mlo, mhi = 2048, 5.0, 3.0e6, 40, 20
    y = _three_laser_links(orc, orbit, t0, dt, N)
    yd = torch.from_numpy(y).cuda()
    out = {}
    for nested in (0, 1):
        tdi = torch.empty((1, 3, N), dtype=torch.float64, device="cuda")
        lib.tdi2(1, N, t0, dt, order, 20, 0, mlo, mhi, yd, dict(orbit, nested=nested), tdi)
        torch.cuda.synchronize()
        out[nested] = tdi.cpu().numpy()[0]
        ref = orc.tdi(y, dict(orbit, nested=nested), t0, dt, order, 20, 0, mlo, mhi)[0]
        assert np.max(np.abs(out[nested] - ref)) < 1e-11  # lasers of unit amplitude
    rms = lambda v: np.sqrt((v[:, mlo:N - mhi] ** 2).mean(axis=1))
    floor = 2e-12 if order == 31 else 1e-6
    assert np.all(rms(out[1]) < floor)
    if order == 31:
        assert np.all(rms(out[0]) > 1e4 * rms(out[1]))


def test_laser_helper_uses_the_travel_time_model(lib, orc):
    N, dt, order, margin = 1 << 12, 5.0, 31, 40
    orbit = dict(synth.kepler_orbit(), tt_order=1)
    p = synth.laser_stream(N)
    yref = orc.laser_links(p, orbit, 0.0, dt, order, margin)
    y = torch.empty((6, N), dtype=torch.float64, device="cuda")
    lib.laser_links(N, 0.0, dt, order, margin, torch.from_numpy(p).cuda(), orbit, y)
    torch.cuda.synchronize()
    rms = np.sqrt(np.mean(yref ** 2))
    assert np.max(np.abs(y.cpu().numpy() - yref)) < 1e-11 * rms
    y0 = orc.laser_links(p, dict(orbit, tt_order=0), 0.0, dt, order, margin)
    assert np.max(np.abs(y0 - yref)) > 1e-6 * rms  # and it matters


def test_static_orbit_ignores_the_delay_model(lib):
    B, N = 2, 4096
    inp = synth.make_inputs(1, B=B, N=N)
    y = torch.randn((B, 6, N), dtype=torch.float64, device="cuda")
    a = torch.empty((B, 3, N), dtype=torch.float64, device="cuda")
    b = torch.empty_like(a)
    lib.tdi2(B, N, 0.0, inp["dt"], 31, 20, 1, inp["margin_lo"], inp["margin_hi"], y, inp["orbit"], a)
    lib.tdi2(B, N, 0.0, inp["dt"], 31, 20, 1, inp["margin_lo"], inp["margin_hi"], y,
             dict(inp["orbit"], tt_order=1, nested=1), b)
    torch.cuda.synchronize()
    assert float((a - b).abs().max()) <= 1e-12 * float(a.abs().max())


def test_bad_delay_model_is_rejected(lib):
    N = 4096
    y = torch.zeros((1, 6, N), dtype=torch.float64, device="cuda")
    out = torch.zeros((1, 3, N), dtype=torch.float64, device="cuda")
    for bad in (dict(tt_order=2), dict(nested=3), dict(tt_order=-1)):
        with pytest.raises(lib.LisaTdError):
            lib.tdi2(1, N, 0.0, 5.0, 31, 20, 1, 160, 144, y, dict(synth.kepler_orbit(), **bad), out)
