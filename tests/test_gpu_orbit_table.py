"""GPU parity on tabulated orbits (kind TABLE, reading A21): the table is sampled
from the oracle's KEPLER1 orbit (the paper's ESA orbit file is not available) and handed, as
the same bits, to both sides."""
import numpy as np
import pytest
import torch

from paper_2501_08261_b200 import synth

pytestmark = pytest.mark.gpu
H_TAB = 86400.0


@pytest.fixture(scope="module")
def lib():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2501_08261_b200 import lib as L
    L.load()
    return L


def _table_orbit(orc, t_lo, t_hi, order=7, h=H_TAB):
    kep = synth.kepler_orbit()
    n_tab = int(np.ceil((t_hi - t_lo) / h)) + 1 + order
    t0 = t_lo - (order // 2) * h
    tab = np.stack([orc.orbit_eval(kep, t0 + h * j)[0] for j in range(n_tab)])
    return {"kind": "table", "r_tab": tab, "t_tab0": t0, "dt_tab": h, "tab_order": order}


@pytest.mark.parametrize("order,t0", [(7, 0.0), (3, 2.5e6)])
def test_chain_on_table_orbit(lib, orc, order, t0):
    B, N = 3, 1 << 14
    inp = synth.make_inputs(3, B=B, N=N)
    dt = inp["dt"]
    orbit = _table_orbit(orc, t0, t0 + N * dt, order, h=H_TAB if order == 7 else 7200.0)
    n = lambda k: None if inp[k] is None else inp[k].numpy()
    ref = orc.chain(inp["l"], inp["m"], n("amp"), n("phase"), n("iota"), n("phi"), n("psi"), n("lam"), n("beta_sky"),
                    orbit, t0, dt, inp["order"], inp["margin_y"], 20, 1, inp["margin_lo"], inp["margin_hi"],
                    alpha=n("alpha"), beta=n("beta"), gamma=n("gamma"), want=("y", "tdi"))
    d = lambda k: None if inp[k] is None else inp[k].cuda()
    hp = torch.empty((B, N), dtype=torch.float64, device="cuda")
    hc = torch.empty_like(hp)
    y = torch.empty((B, 6, N), dtype=torch.float64, device="cuda")
    tdi = torch.empty((B, 3, N), dtype=torch.float64, device="cuda")
    lib.modes_to_pol(B, N, inp["l"], inp["m"], d("amp"), d("phase"), d("alpha"), d("beta"), d("gamma"), d("iota"),
                     d("phi"), d("psi"), None, hp, hc)
    lib.link_response(B, N, t0, dt, inp["order"], inp["margin_y"], hp, hc, d("lam"), d("beta_sky"), orbit, y)
    lib.tdi2(B, N, t0, dt, inp["order"], 20, 1, inp["margin_lo"], inp["margin_hi"], y, orbit, tdi)
    torch.cuda.synchronize()
    yg, tg = y.cpu().numpy(), tdi.cpu().numpy()
    for b in range(B):
        for l in range(6):
            err = np.linalg.norm(yg[b, l] - ref["y"][b, l]) / np.linalg.norm(ref["y"][b, l])
            assert err < 5e-13, (b, l, err)
        common = max(np.linalg.norm(ref["tdi"][b, c]) for c in range(3))
        errs = [np.linalg.norm(tg[b, c] - ref["tdi"][b, c]) / common for c in range(3)]
        print("table orbit walker", b, errs)
        assert max(errs) < 1e-11


def test_laser_links_and_generic_tdi_on_table_orbit(lib, orc):
    N, dt, order, margin = 1 << 13, 5.0, 7, 32
    orbit = _table_orbit(orc, 0.0, N * dt)
    p = synth.laser_stream(N)
    yref = orc.laser_links(p, orbit, 0.0, dt, order, margin)
    y = torch.empty((6, N), dtype=torch.float64, device="cuda")
    lib.laser_links(N, 0.0, dt, order, margin, torch.from_numpy(p).cuda(), orbit, y)
    torch.cuda.synchronize()
    rms = np.sqrt(np.mean(yref ** 2))
    assert np.max(np.abs(y.cpu().numpy() - yref)) < 1e-11 * rms
    mlo, mhi = margin + 20, margin + 8
    ref = orc.tdi(yref[None], orbit, 0.0, dt, order, 20, 0, mlo, mhi)
    out = torch.empty((1, 3, N), dtype=torch.float64, device="cuda")
    lib.tdi2(1, N, 0.0, dt, order, 20, 0, mlo, mhi, y.view(1, 6, N), orbit, out)   # order 7: generic kernel
    torch.cuda.synchronize()
    assert np.max(np.abs(out.cpu().numpy() - ref)) < 1e-11 * rms


def test_table_must_cover_the_grid(lib, orc):
    N = 4096
    orbit = _table_orbit(orc, 0.0, N * 5.0)
    z = torch.zeros((1, N), dtype=torch.float64, device="cuda")
    y = torch.zeros((1, 6, N), dtype=torch.float64, device="cuda")
    with pytest.raises(lib.LisaTdError) as e:
        lib.link_response(1, N, 1.0e7, 5.0, 31, 128, z, z, z[0, :1], z[0, :1], orbit, y)
    assert "does not cover" in str(e.value)


def test_table_orbit_outside_the_host_bounds_is_reported_not_clamped(lib, orc):
    """The kernels size their shared-memory tiles from host-side bounds on the orbit; for a TABLE orbit
    those come from its nodes (chord rates x 1.05).  A table whose centroid swings by +-1.2e11 m from one
    hourly node to the next is interpolated with a peak rate 1.29 times the chord rate: the common
    delay drifts across a 256-sample tile by more samples than the strain tile has halo for.  The kernel
    must say so (sticky flag -> LISA_TD_EINVAL at the next lisa_td_check), not clamp and carry on."""
    B, N, dt, t0, h, q = 2, 1 << 14, 5.0, 1.0e6, 3600.0, 7
    kep = synth.kepler_orbit()
    n_tab = int(np.ceil(N * dt / h)) + 2 + 2 * q
    t_tab0 = t0 - q * h
    tab = np.stack([orc.orbit_eval(kep, t_tab0 + h * j)[0] for j in range(n_tab)])
    good = {"kind": "table", "r_tab": tab.copy(), "t_tab0": t_tab0, "dt_tab": h, "tab_order": q}
    wild = tab.copy()
    wild[::2, :, 0] += 1.2e11
    wild[1::2, :, 0] -= 1.2e11
    bad = {"kind": "table", "r_tab": wild, "t_tab0": t_tab0, "dt_tab": h, "tab_order": q}
    rng = np.random.default_rng(0)
    hp = torch.from_numpy(rng.standard_normal((B, N))).cuda()
    hc = torch.from_numpy(rng.standard_normal((B, N))).cuda()
    lam = torch.tensor([0.3, 2.0], dtype=torch.float64, device="cuda")
    bet = torch.tensor([0.1, -0.2], dtype=torch.float64, device="cuda")
    y = torch.empty((B, 6, N), dtype=torch.float64, device="cuda")
    lib.link_response(B, N, t0, dt, 31, 300, hp, hc, lam, bet, good, y)
    lib.check()                                   # a sane table raises nothing
    lib.link_response(B, N, t0, dt, 31, 300, hp, hc, lam, bet, bad, y)
    with pytest.raises(lib.LisaTdError) as e:
        lib.check()
    assert e.value.code == -1 and "link-response" in str(e.value)
    lib.check()                                   # the flag is cleared by the check that reported it
