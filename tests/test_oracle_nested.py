"""Pins of the oracle's delay model of reading A22:
first-order light travel times L_l = (d/c)(1 + n.v_s/c) and TDI delays chained along the light
path (oracle/lisa_oracle.c orbit_state, orbit_eval, nested_delay, X15_NESTED, X20_NESTED)."""
import numpy as np
import pytest

from paper_2501_08261_b200 import synth

C_LIGHT = 299792458.0
S = [3, 1, 2, 2, 3, 1]  # sender / receiver of links [1,2,3,-1,-2,-3]
R = [2, 3, 1, 3, 1, 2]


def _idx(label):
    return label - 1 if label > 0 else -label + 2


def _daily_table(orc, t_lo, t_hi):
    kep = synth.kepler_orbit()
    h = 86400.0
    t_tab = t_lo - 5 * h + h * np.arange(int((t_hi - t_lo) / h) + 12)
    tab = np.stack([orc.orbit_eval(kep, float(t))[0] for t in t_tab])
    return {"kind": "table", "r_tab": tab, "t_tab0": float(t_tab[0]), "dt_tab": h, "tab_order": 7}


def _exact_travel_time(orc, orbit, link, t):
    """fixed point of c L = |r_r(t) - r_s(t - L)| from the positions alone"""
    pos = dict(orbit, tt_order=0, nested=0)
    rr = orc.orbit_state(pos, t)[0][R[link] - 1]
    L = 8.0
    for _ in range(8):
        rs = orc.orbit_state(pos, t - L)[0][S[link] - 1]
        L = np.linalg.norm(rr - rs) / C_LIGHT
    return L


@pytest.mark.parametrize("kind", ["kepler1", "table"])
def test_velocity_is_the_time_derivative_of_the_position(orc, kind):
    orbit = synth.kepler_orbit() if kind == "kepler1" else _daily_table(orc, 0.0, 3.0e6)
    for t in (1.0e5 + 17.0, 1.234e6, 2.9e6):
        r, v = orc.orbit_state(orbit, t)
        h = 20.0
        fd = (orc.orbit_state(orbit, t + h)[0] - orc.orbit_state(orbit, t - h)[0]) / (2 * h)
        # positions are returned in fp64 (ulp(1.5e11 m) = 3e-5 m): fd is good to ~2e-6 m/s
        assert np.max(np.abs(v - fd)) < 1e-5
        assert 2.9e4 < np.max(np.linalg.norm(v, axis=1)) < 3.1e4  # orbital speed ~ 29.8 km/s
    r, v = orc.orbit_state(synth.static_orbit(), 5.0)
    assert np.all(v == 0.0)


def test_first_order_travel_time_against_the_fixed_point(orc):
    """tt_order 1 is the solution of c L = |r_r(t) - r_s(t - L)| up to O(v^2/c^2) ~ 1e-8 relative;
    tt_order 0 misses it by up to ~8e-4 s, with opposite signs for l and -l"""
    kep = synth.kepler_orbit()
    worst0 = 0.0
    for t in (0.0, 2.5e6, 7.7e6, 1.9e7):
        L0 = orc.orbit_eval(dict(kep, tt_order=0), t)[1]
        L1 = orc.orbit_eval(dict(kep, tt_order=1), t)[1]
        for l in range(6):
            Lx = _exact_travel_time(orc, kep, l, t)
            assert abs(L1[l] - Lx) < 2e-7
            worst0 = max(worst0, abs(L0[l] - Lx))
        for a in range(3):  # tt_order 0 is symmetric, tt_order 1 is not (Sagnac-like split)
            assert L0[a] == L0[a + 3]
            assert (L1[a] - L0[a]) * (L1[a + 3] - L0[a + 3]) < 0
    assert 1e-4 < worst0 < 2e-3
    st = synth.static_orbit()
    assert np.array_equal(orc.orbit_eval(dict(st, tt_order=1), 3.0)[1], orc.orbit_eval(st, 3.0)[1])


def test_nested_delay_follows_the_light_path(orc):
    """the chained delay of labels l_0, l_1, ... equals the travel time of light traced back leg by
    leg (exact fixed point per leg) through spacecraft R[l_0] <- S[l_0] = R[l_1] <- ..."""
    kep = dict(synth.kepler_orbit(), tt_order=1)
    for labels in ([3, -3, -2, 2, -2, 2, 3], [-2, 2, 3, -3, 3, -3, -2], [1, -1, -3, 3], [2]):
        for i in range(len(labels) - 1):  # the legs connect
            assert S[_idx(labels[i])] == R[_idx(labels[i + 1])]
        t = 4.4e6
        tau = 0.0
        for lab in labels:
            tau += _exact_travel_time(orc, kep, _idx(lab), t - tau)
        got = orc.nested_delay(kep, t, labels)
        assert abs(got - tau) < 2e-7 * len(labels)
        # summed at the output time instead: off by ~ tau * dL/dt
        summed = sum(orc.orbit_eval(kep, t)[1][_idx(lab)] for lab in labels)
        if len(labels) > 1:
            assert abs(summed - got) > 1e-8
        else:
            assert summed == got
    assert orc.nested_delay(kep, 1.0e6, []) == 0.0


@pytest.mark.parametrize("generation", [15, 20])
def test_nested_equals_summed_on_a_static_constellation(orc, generation):
    rng = np.random.default_rng(7)
    N = 400
    y = rng.standard_normal((2, 6, N))
    st = synth.static_orbit()
    st["L_static"] = [8.1, 8.3, 8.2, 8.15, 8.35, 8.25]  # unequal, constant
    a = orc.tdi(y, dict(st, nested=0), 0.0, 5.0, 7, generation, 0, 40, 8)
    b = orc.tdi(y, dict(st, nested=1), 0.0, 5.0, 7, generation, 0, 40, 8)
    scale = np.abs(a).max()
    assert np.max(np.abs(a - b)) < 1e-15 * scale  # same delays up to the order of the additions


def _three_laser_links(orc, orbit, t0, dt, N):
    """y_slr(t_n) = p_s(t_n - L_l(t_n)) - p_r(t_n) for three analytic lasers (no interpolation)"""
    f = np.array([3.1e-3, 4.7e-3, 6.3e-3], dtype=np.longdouble)
    ph = np.array([0.3, 1.1, 2.5], dtype=np.longdouble)
    t = np.longdouble(t0) + np.arange(N, dtype=np.longdouble) * np.longdouble(dt)
    L = np.array([orc.orbit_eval(orbit, float(tt))[1] for tt in t]).astype(np.longdouble)
    p = lambda i, tt: np.sin(2 * np.pi * f[i] * tt + ph[i])
    y = np.zeros((1, 6, N))
    for l in range(6):
        y[0, l] = (p(S[l] - 1, t - L[:, l]) - p(R[l] - 1, t)).astype(np.float64)
    return y


def test_chained_generation_2_cancels_three_lasers_on_flexing_arms(orc):
    """'TDI 2 beats TDI 1.5 on flexing arms' holds only with chained delays in the order
    of the light path.  Three independent unit-amplitude lasers on KEPLER1 arms with first-order
    travel times (L_l != L_-l): chained X2,Y2,Z2 cancel them to the interpolation/rounding floor
    (~1e-13); chained generation 1.5, and generation 2 with delays summed at the output time
    (reading A10), leave ~1e-8.  One transposed or mislabelled delay in X20_NESTED costs 5 orders."""
    orbit = dict(synth.kepler_orbit(), tt_order=1)
    N, dt, t0, order, mlo, mhi = 1536, 5.0, 3.0e6, 31, 40, 20
    y = _three_laser_links(orc, orbit, t0, dt, N)
    rms = {}
    for nested in (0, 1):
        for gen in (15, 20):
            X = orc.tdi(y, dict(orbit, nested=nested), t0, dt, order, gen, 0, mlo, mhi)
            rms[nested, gen] = np.sqrt((X[0][:, mlo:N - mhi] ** 2).mean(axis=1))
    assert np.all(rms[1, 20] < 2e-12)
    assert np.all(rms[1, 15] > 1e4 * rms[1, 20])
    assert np.all(rms[0, 20] > 1e4 * rms[1, 20])
    # travel-time model of the TDI delays must be the one the links were built with
    X = orc.tdi(y, dict(orbit, nested=1, tt_order=0), t0, dt, order, 20, 0, mlo, mhi)
    assert np.all(np.sqrt((X[0][:, mlo:N - mhi] ** 2).mean(axis=1)) > 1e3 * rms[1, 20])


def test_three_laser_links_helper_matches_the_analytic_links(orc):
    """orc_laser_links3 (sampled lasers, fractional-delay reads) against the analytic construction"""
    orbit = dict(synth.kepler_orbit(), tt_order=1)
    N, dt, t0 = 512, 5.0, 1.0e6
    want = _three_laser_links(orc, orbit, t0, dt, N)[0]
    f = np.array([3.1e-3, 4.7e-3, 6.3e-3], dtype=np.longdouble)
    ph = np.array([0.3, 1.1, 2.5], dtype=np.longdouble)
    t = np.longdouble(t0) + np.arange(N, dtype=np.longdouble) * np.longdouble(dt)
    p3 = np.stack([np.sin(2 * np.pi * f[i] * t + ph[i]) for i in range(3)]).astype(np.float64)
    got = orc.laser_links3(p3, orbit, t0, dt, 31, 24)
    assert np.all(got[:, :24] == 0.0) and np.all(got[:, N - 24:] == 0.0)
    assert np.max(np.abs(got[:, 24:N - 24] - want[:, 24:N - 24])) < 1e-12
