"""C11 of SURVEY.md section 8(c) (reading A12) and the pin of orc_laser_links.

A common laser p(t) injected at link level, y_l(t) = p(t - L_l(t)) - p(t), cancels in the Michelson
combinations only if the arms are static.  With the delays of Eq. 2.9 / 2.10 SUMMED and every L_l
taken at the output time (reading A10), a term  s y_l(t - D)  reads
p(t - D - L_l(t - D)) with L_l(t - D) = L_l(t) - Ldot_l D + ..., so to first order in the arm rates

    X_res(t) = sum_terms  s * Ldot_l(t) * D(t) * pdot(t - D - L_l)                          (*)

(the zeroth order cancels identically).  For slowly varying p the sum collapses to

    X1.5_res = pdot(t) [ (L2 + L-2)(Ldot3 + Ldot-3) - (L3 + L-3)(Ldot2 + Ldot-2) ]           (**)
    |X2_res| = 2 (L2 + L-2 + L3 + L-3) omega |X1.5_res| = 8 omega L |X1.5_res|   (equal-ish arms),

the "factor the equations imply" of BASELINE.json's north_star.  The oracle's measured residual
(orc_laser_links -> orc_tdi, KEPLER1 arms, order 31) must follow (*) to 1e-5 of the largest channel and (**) to a few per
cent at 0.05-0.1 mHz.  A wrong delay label, sign or evaluation time in the term tables, or link noise
built with the wrong arm, changes (*) at order one.
"""
import math
import os

import numpy as np
import pytest

from paper_2501_08261_b200 import synth

LINKS = [1, 2, 3, -1, -2, -3]
GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "tdi_terms.txt")


def lidx(link):
    return link - 1 if link > 0 else -link + 2


def cyc(link, times):
    a = abs(link)
    for _ in range(times):
        a = a % 3 + 1
    return a if link > 0 else -a


def load_terms(tag):
    terms = []
    for line in open(GOLDEN):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        head, _, tail = line.partition(":")
        g, sign, link = head.split()
        if g == tag:
            terms.append((1 if sign == "+" else -1, int(link), [int(x) for x in tail.split()]))
    return terms


class Laser:
    """band-limited analytic laser phase: p(t) = sum a_i sin(w_i t + phi_i)"""

    def __init__(self, rng, freqs):
        self.w = 2 * math.pi * np.asarray(freqs)
        self.a = rng.uniform(0.5, 1.5, len(freqs)) * 1e-13
        self.ph = rng.uniform(0, 2 * math.pi, len(freqs))

    def p(self, t):
        return np.sum(self.a[:, None] * np.sin(self.w[:, None] * t[None, :] + self.ph[:, None]), axis=0)

    def pdot(self, t):
        return np.sum((self.a * self.w)[:, None] * np.cos(self.w[:, None] * t[None, :] + self.ph[:, None]), axis=0)


def arm_times_and_rates(orc, orbit, t, h=2000.0):
    """L_l, dL_l/dt, d2L_l/dt2 at the times t ([N][6] each) by central differences of orc_orbit_eval"""
    L = np.array([orc.orbit_eval(orbit, ti)[1] for ti in t])
    Lp = np.array([orc.orbit_eval(orbit, ti + h)[1] for ti in t])
    Lm = np.array([orc.orbit_eval(orbit, ti - h)[1] for ti in t])
    return L, (Lp - Lm) / (2 * h), (Lp - 2 * L + Lm) / (h * h)


def first_order_residual(terms, c, L, Ld, Ldd, laser, t):
    """(*) with the arm at the delayed time expanded one order further, L_l(t - D) = L_l - Ldot_l D +
    Lddot_l D^2 / 2: the curvature term matters at low frequency, where (*) itself falls like omega"""
    res = np.zeros_like(t)
    for sign, link, labels in terms:
        D = sum(L[:, lidx(cyc(lab, c))] for lab in labels) if labels else np.zeros_like(t)
        l = lidx(cyc(link, c))
        res += sign * (Ld[:, l] * D - 0.5 * Ldd[:, l] * D * D) * laser.pdot(t - D - L[:, l])
    return res


@pytest.mark.parametrize("gen", [15, 20])
def test_c11_first_order_laser_residual(orc, gen):
    rng = np.random.default_rng(gen)
    N, dt, order, t0, margin = 2048, 5.0, 31, 4.0e6, 32
    orbit = synth.kepler_orbit()
    laser = Laser(rng, [0.6e-3, 0.9e-3, 2.3e-3, 4.1e-3])
    t = t0 + np.arange(N) * dt
    y = orc.laser_links(laser.p(t), orbit, t0, dt, order, margin)
    mlo, mhi = margin + 32, margin + 16
    xyz = orc.tdi(y[None], orbit, t0, dt, order, gen, 0, mlo, mhi)[0]
    sl = slice(mlo + 8, N - mhi - 8, 16)
    L, Ld, Ldd = arm_times_and_rates(orc, orbit, t[sl])
    terms = load_terms(str(gen))
    rms_y = np.sqrt(np.mean(y[:, margin:-margin] ** 2))
    refs = [first_order_residual(terms, c, L, Ld, Ldd, laser, t[sl]) for c in range(3)]
    # p enters as doubles: its 1e-16 white rounding does not cancel in TDI and sits 1e-6..1e-4 below a
    # residual that is itself 1e-7 of the link noise, so the three channels are held to their common scale
    scale = max(np.linalg.norm(r) for r in refs)
    for c in range(3):
        err = np.linalg.norm(xyz[c, sl] - refs[c]) / scale
        assert err < 1e-5, (gen, c, err)
        assert np.linalg.norm(refs[c]) > 0.03 * scale
    # the residual is a ~1e-7 remnant of the link noise: the check is about a small quantity
    assert 1e-9 < scale / np.sqrt(len(refs[0])) / rms_y < 1e-5


def test_c11_low_frequency_limit_and_generation_ratio(orc):
    rng = np.random.default_rng(3)
    N, dt, order, t0, margin = 8192, 5.0, 31, 1.0e6, 32
    orbit = synth.kepler_orbit()
    f = 0.07e-3
    laser = Laser(rng, [f])
    t = t0 + np.arange(N) * dt
    y = orc.laser_links(laser.p(t), orbit, t0, dt, order, margin)
    mlo, mhi = margin + 32, margin + 16
    x15 = orc.tdi(y[None], orbit, t0, dt, order, 15, 0, mlo, mhi)[0, 0]
    x20 = orc.tdi(y[None], orbit, t0, dt, order, 20, 0, mlo, mhi)[0, 0]
    sl = slice(mlo + 8, N - mhi - 8, 64)
    L, Ld, _ = arm_times_and_rates(orc, orbit, t[sl])
    i2, m2, i3, m3 = lidx(2), lidx(-2), lidx(3), lidx(-3)
    K = (L[:, i2] + L[:, m2]) * (Ld[:, i3] + Ld[:, m3]) - (L[:, i3] + L[:, m3]) * (Ld[:, i2] + Ld[:, m2])
    ref = K * laser.pdot(t[sl])
    # corrections are O(omega x 4L) = 1.5 % at 0.07 mHz
    assert np.linalg.norm(x15[sl] - ref) / np.linalg.norm(ref) < 0.03
    # generation 2 on un-nested delays: larger residual relative to X1.5 by 2 omega (L2+L-2+L3+L-3)
    ratio = np.sqrt(np.mean(x20[sl] ** 2) / np.mean(x15[sl] ** 2))
    implied = 2 * (2 * math.pi * f) * np.mean(L[:, i2] + L[:, m2] + L[:, i3] + L[:, m3])
    assert abs(ratio / implied - 1) < 0.03
    # on STATIC arms of the same size both residuals vanish (interpolation error only)
    st = synth.static_orbit()
    ys = orc.laser_links(laser.p(t), st, t0, dt, order, margin)
    for gen in (15, 20):
        xs = orc.tdi(ys[None], st, t0, dt, order, gen, 0, mlo, mhi)[0]
        assert np.max(np.abs(xs)) < 1e-6 * np.sqrt(np.mean(x15[sl] ** 2))


@pytest.mark.parametrize("kind,tt_order", [("static", 0), ("kepler1", 0), ("kepler1", 1)])
def test_laser_links_is_laser_links3_with_one_laser(orc, kind, tt_order):
    """orc_laser_links (one common laser) against orc_laser_links3 (three lasers, pinned by analytic
    lasers and three-laser cancellation in test_oracle_nested.py) fed the same stream three times,
    and against the definition y_l[n] = p(n - L_l(t_n)/dt) - p[n] read with orc_delay_read."""
    rng = np.random.default_rng(7)
    N, dt, order, t0, margin = 700, 5.0, 31, 2.0e6, 40
    orbit = dict(synth.static_orbit() if kind == "static" else synth.kepler_orbit(), tt_order=tt_order)
    p = rng.standard_normal(N)
    y1 = orc.laser_links(p, orbit, t0, dt, order, margin)
    y3 = orc.laser_links3(np.stack([p, p, p]), orbit, t0, dt, order, margin)
    assert np.array_equal(y1, y3)
    assert np.all(y1[:, :margin] == 0) and np.all(y1[:, N - margin:] == 0)
    for n in (margin, 123, 356, N - margin - 1):
        Ls = orc.orbit_eval(orbit, t0 + n * dt)[1]
        for l in range(6):
            want = orc.delay_read(p, n, Ls[l] / dt, order) - p[n]
            assert abs(y1[l, n] - want) < 1e-14
    # three DIFFERENT lasers do change the answer (the comparison above is not vacuous)
    q = rng.standard_normal(N)
    assert np.max(np.abs(orc.laser_links3(np.stack([p, q, p]), orbit, t0, dt, order, margin) - y1)) > 0.1
