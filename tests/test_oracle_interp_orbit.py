"""Pins of the oracle's fractional-delay read (O-I, C8) and of its orbit model (reading A8)."""
import math

import numpy as np
import pytest

from paper_2501_08261_b200 import synth


@pytest.mark.parametrize("order", [1, 3, 7, 31])
def test_lagrange_partition_of_unity_and_nodes(orc, order):
    for eps in (0.0, 0.1, 0.5, 0.93):
        c = orc.lagrange_coeffs(order, eps)
        assert abs(np.sum(c) - 1.0) < 1e-14
    h = (order + 1) // 2
    c0 = orc.lagrange_coeffs(order, 0.0)  # eps = 0 -> the tap j = 0 itself
    expect = np.zeros(order + 1)
    expect[h - 1] = 1.0
    assert np.max(np.abs(c0 - expect)) < 1e-15


@pytest.mark.parametrize("order", [1, 3, 7, 31])
def test_delay_read_exact_on_polynomials(orc, order):
    # a degree-p polynomial is reproduced exactly by the (p+1)-tap interpolant
    N = 256
    n = np.arange(N, dtype=np.float64)
    rng = np.random.default_rng(order)
    deg = min(order, 9)  # keep values well-conditioned in fp64 input
    coef = rng.uniform(-1, 1, deg + 1)
    z = (n - 128.0) / 32.0
    x = np.polyval(coef, z)
    for D in (0.0, 3.0, 0.37, 7.81, -4.25, 11.999):
        got = orc.delay_read(x, 128, D, order)
        ref = np.polyval(coef, (128.0 - D - 128.0) / 32.0)
        assert abs(got - ref) < 2e-13 * np.max(np.abs(x)), (order, D)


def test_delay_read_linear_is_paper_interpolation(orc):
    # order 1 = the paper's linear interpolation
    x = np.random.default_rng(0).standard_normal(64)
    D = 2.3  # between samples n-3 and n-2
    got = orc.delay_read(x, 40, D, 1)
    assert abs(got - (0.3 * x[37] + 0.7 * x[38])) < 1e-15


def test_delay_read_zero_extension_and_integer(orc):
    x = np.arange(1.0, 33.0)
    assert orc.delay_read(x, 10, 4.0, 31) == x[6]
    assert orc.delay_read(x, 2, 5.0, 31) == 0.0  # outside the grid
    # window partly outside: equals the same read on an explicitly zero-padded series
    xp = np.concatenate([np.zeros(40), x, np.zeros(40)])
    assert abs(orc.delay_read(x, 5, 2.5, 31) - orc.delay_read(xp, 45, 2.5, 31)) < 1e-15


def test_static_orbit_is_equilateral(orc):
    o = synth.static_orbit()
    r, L = orc.orbit_eval(o, 123.0)
    for i in range(3):
        j = (i + 1) % 3
        assert abs(np.linalg.norm(r[i] - r[j]) - synth.ARM) < 1e-5
    assert np.allclose(L, synth.ARM / synth.C_LIGHT, rtol=0, atol=1e-15)
    assert np.max(np.abs(np.sum(r, axis=0))) < 1e-5  # centred on the origin


def test_kepler1_orbit_invariants(orc):
    o = synth.kepler_orbit()
    a, L = synth.AU, synth.ARM
    delta = L / (2 * a)
    e = math.sqrt(1 + 2 * delta / math.sqrt(3) + 4 * delta ** 2 / 3) - 1
    inc = math.atan(delta / (1 + delta / math.sqrt(3)))
    assert abs(e - 0.004859) < 2e-6  # SURVEY A8 scratch value
    ts = np.linspace(0.0, synth.YEAR, 97)
    arms = []
    for t in ts:
        r, Lt = orc.orbit_eval(o, t)
        for k in range(3):
            d = np.linalg.norm(r[k])
            assert a * (1 - e) * (1 - 1e-6) <= d <= a * (1 + e) * (1 + 1e-6)  # Kepler ellipse radii
        # light travel time = geometric distance / c; L_l = L_{-l}
        assert np.allclose(Lt[:3], Lt[3:], rtol=0, atol=1e-15)
        assert abs(Lt[0] * synth.C_LIGHT - np.linalg.norm(r[1] - r[2])) < 1e-3  # link 1: 3 -> 2
        assert abs(Lt[1] * synth.C_LIGHT - np.linalg.norm(r[2] - r[0])) < 1e-3  # link 2: 1 -> 3
        assert abs(Lt[2] * synth.C_LIGHT - np.linalg.norm(r[0] - r[1])) < 1e-3  # link 3: 2 -> 1
        arms.extend(Lt[:3] * synth.C_LIGHT)
    arms = np.array(arms)
    # time-varying unequal arms with ~1 % breathing around 2.5e9 m (2.495-2.524e9)
    assert 2.49e9 < arms.min() < 2.50e9 and 2.52e9 < arms.max() < 2.53e9
    # each spacecraft's orbit is planar, inclined by inc to the ecliptic, normal fixed in time
    r0, _ = orc.orbit_eval(o, 0.0)
    r1, _ = orc.orbit_eval(o, 0.21 * synth.YEAR)
    r2, _ = orc.orbit_eval(o, 0.57 * synth.YEAR)
    for k in range(3):
        nrm = np.cross(r0[k], r1[k])
        nrm /= np.linalg.norm(nrm)
        assert abs(np.dot(nrm, r2[k])) / a < 1e-12
        assert abs(math.acos(abs(nrm[2])) - inc) < 1e-9
    # spacecraft 2 is spacecraft 1 a third of a year earlier, rotated by 120 degrees about z
    t = 0.3 * synth.YEAR
    ra, _ = orc.orbit_eval(o, t)
    rb, _ = orc.orbit_eval(o, t - synth.YEAR / 3)
    c, s = math.cos(2 * math.pi / 3), math.sin(2 * math.pi / 3)
    rot = np.array([[c, -s, 0], [s, c, 0], [0, 0, 1]])
    assert np.max(np.abs(ra[1] - rot @ rb[0])) / a < 1e-13


def test_kepler1_solves_kepler_equation_to_first_order(orc):
    # psi = M + e sin M solves psi - e sin psi = M up to O(e^2): position differs from the exact
    # Kepler position by less than ~ a e^2
    o = synth.kepler_orbit()
    a = synth.AU
    delta = synth.ARM / (2 * a)
    e = math.sqrt(1 + 2 * delta / math.sqrt(3) + 4 * delta ** 2 / 3) - 1
    inc = math.atan(delta / (1 + delta / math.sqrt(3)))
    for t in (0.0, 1e6, 7.7e6, 2.1e7):
        r, _ = orc.orbit_eval(o, t)
        M = 2 * math.pi * t / synth.YEAR
        E = M
        for _ in range(50):
            E = M + e * math.sin(E)
        exact = np.array([a * (math.cos(E) - e) * math.cos(inc), a * math.sqrt(1 - e * e) * math.sin(E),
                          a * (math.cos(E) - e) * math.sin(inc)])
        assert np.linalg.norm(r[0] - exact) < 1.5 * a * e * e
