"""Pins of the oracle's tabulated-orbit kind (oracle/lisa_oracle.c orbit_eval kind 2; PAPER.md:134,
reading A21 of DESIGN.md)."""
import numpy as np

from paper_2501_08261_b200 import synth

C_LIGHT = 299792458.0


def _table_from(fn, t_tab):
    return np.stack([fn(t) for t in t_tab])


def test_polynomial_trajectories_are_reproduced_exactly(orc):
    """degree <= tab_order polynomials in t are reproduced to rounding, anywhere in the table,
    including the clamped first and last intervals"""
    rng = np.random.default_rng(0)
    q, n_tab, t0, h = 7, 20, -3.0e5, 86400.0
    coef = rng.standard_normal((q + 1, 3, 3)) * 1e9
    poly = lambda t: sum(coef[m] * ((t - t0) / (n_tab * h)) ** m for m in range(q + 1))
    t_tab = t0 + h * np.arange(n_tab)
    orbit = {"kind": "table", "r_tab": _table_from(poly, t_tab), "t_tab0": t0, "dt_tab": h, "tab_order": q}
    for t in [t0 + 10.0, t0 + 0.4 * h, t0 + 7.77 * h, t0 + 18.9 * h, t0 + 12 * h]:
        r, L = orc.orbit_eval(orbit, t)
        want = poly(t)
        assert np.max(np.abs(r - want)) < 1e-12 * np.max(np.abs(want))
        S, R = [3, 1, 2, 2, 3, 1], [2, 3, 1, 3, 1, 2]
        for k in range(6):
            assert abs(L[k] - np.linalg.norm(want[R[k] - 1] - want[S[k] - 1]) / C_LIGHT) < 1e-13 * L[k]


def test_table_nodes_are_returned_at_the_nodes(orc):
    rng = np.random.default_rng(1)
    tab = rng.standard_normal((12, 3, 3)) * 1e10
    orbit = {"kind": "table", "r_tab": tab, "t_tab0": 100.0, "dt_tab": 50.0, "tab_order": 3}
    for j in (0, 1, 5, 10, 11):
        r, _ = orc.orbit_eval(orbit, 100.0 + 50.0 * j)
        assert np.max(np.abs(r - tab[j])) <= 1e-15 * np.max(np.abs(tab[j]))


def test_kepler1_table_matches_kepler1_closed_form(orc):
    """a daily table of the analytic orbit, interpolated at degree 7, agrees with the analytic
    orbit to ~1e-6 m (interpolation error a (w h)^8 / 8! x node factor), i.e. 3e-15 s of delay"""
    kep = synth.kepler_orbit()
    h = 86400.0
    t_tab = -4 * h + h * np.arange(80)
    tab = _table_from(lambda t: orc.orbit_eval(kep, t)[0], t_tab)
    orbit = {"kind": "table", "r_tab": tab, "t_tab0": float(t_tab[0]), "dt_tab": h, "tab_order": 7}
    worst = 0.0
    for t in np.linspace(0.0, 60 * h, 97):
        r, L = orc.orbit_eval(orbit, t)
        rk, Lk = orc.orbit_eval(kep, t)
        worst = max(worst, np.max(np.abs(r - rk)))
        assert np.max(np.abs(L - Lk)) < 1e-13
    assert worst < 1e-4, worst


def test_chain_on_kepler1_table_matches_chain_on_kepler1(orc):
    """the whole S1..S3 chain on the tabulated orbit agrees with the chain on the closed-form
    orbit it was sampled from (the two orbit kinds share no code path in orbit_eval)"""
    N = 4096
    inp = synth.make_inputs(3, B=1, N=N)
    kep = inp["orbit"]
    h = 86400.0
    t_tab = -5 * h + h * np.arange(12)
    tab = _table_from(lambda t: orc.orbit_eval(kep, t)[0], t_tab)
    tabo = {"kind": "table", "r_tab": tab, "t_tab0": float(t_tab[0]), "dt_tab": h, "tab_order": 7}
    n = lambda k: None if inp[k] is None else inp[k].numpy()
    run = lambda o: orc.chain(inp["l"], inp["m"], n("amp"), n("phase"), n("iota"), n("phi"), n("psi"), n("lam"),
                              n("beta_sky"), o, inp["t0"], inp["dt"], inp["order"], inp["margin_y"], 20, 1,
                              inp["margin_lo"], inp["margin_hi"], alpha=n("alpha"), beta=n("beta"),
                              gamma=n("gamma"), want=("y", "tdi"))
    a, b = run(kep), run(tabo)
    for l in range(6):
        assert np.linalg.norm(a["y"][0, l] - b["y"][0, l]) / np.linalg.norm(a["y"][0, l]) < 1e-11
    common = max(np.linalg.norm(a["tdi"][0, c]) for c in range(3))
    for c in range(3):
        assert np.linalg.norm(a["tdi"][0, c] - b["tdi"][0, c]) / common < 1e-9
