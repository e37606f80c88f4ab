"""C12 of SURVEY.md section 8(c): a second, deliberately different brute-force evaluation of S2 and S3
on tiny grids, which the oracle (oracle/lisa_oracle.c, long-double build) must reproduce to ~1e-15.

Differences from the oracle, on purpose:
  - delays go through ABSOLUTE times: the read happens at t_eval = t - L - k.r_s/c (Eq. 2.8,
    PAPER.md:149-161) resp. t - sum L_l (Eq. 2.9/2.10), and the p+1 nodes are
    addressed by their absolute times t0 + i dt, instead of the oracle's delay in samples split
    into an integer and a fraction;
  - the interpolating polynomial through the p+1 nodes is evaluated with NEVILLE's recursion, not
    with Lagrange basis products (the interpolant is unique, so the two must agree);
  - numpy long double (x86 80-bit), vectorised over samples, written here from the paper and the
    readings of DESIGN.md section 2 (A7, A8, A10, A11, O-I); the TDI term table is read from
    tests/golden/tdi_terms.txt.
"""
import math
import os

import numpy as np
import pytest

from paper_2501_08261_b200 import synth

LD = np.longdouble
C = LD(synth.C_LIGHT)
LINKS = [1, 2, 3, -1, -2, -3]
SR = {1: (3, 2), 2: (1, 3), 3: (2, 1), -1: (2, 3), -2: (3, 1), -3: (1, 2)}
GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "tdi_terms.txt")

pytestmark = pytest.mark.skipif(np.finfo(LD).eps > 2e-19, reason="needs 80-bit long double")


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


def neville_read(x, t0, dt, order, t_out, t_eval):
    """Value at the absolute times t_eval[n] of the polynomial through the order+1 samples of x
    nearest to it in the sense of O-I: K = ceil((t_out - t_eval)/dt), nodes n - K - h + 1 .. n - K + h
    (h = (order+1)/2), x = 0 outside the grid.  Neville's recursion on absolute node times."""
    N = x.shape[0]
    h = (order + 1) // 2
    n = np.arange(N)
    K = np.ceil((t_out - t_eval) / dt).astype(np.int64)
    first = n - K - h + 1
    idx = first[None, :] + np.arange(order + 1)[:, None]           # [p+1][N]
    ok = (idx >= 0) & (idx < N)
    P = np.where(ok, x[np.clip(idx, 0, N - 1)], LD(0))
    tn = t0 + idx.astype(LD) * dt                                  # absolute node times
    for m in range(1, order + 1):
        for i in range(order + 1 - m):
            P[i] = ((t_eval - tn[i + m]) * P[i] + (tn[i] - t_eval) * P[i + 1]) / (tn[i] - tn[i + m])
    return P[0]


def positions(orbit, t):
    """r[3][3][N] metres (reading A8 for KEPLER1), long double."""
    N = t.shape[0]
    r = np.zeros((3, 3, N), dtype=LD)
    if orbit["kind"] == "static":
        for k in range(3):
            for j in range(3):
                r[k, j] = LD(orbit["r_static"][k][j])
        return r
    a, Lm, yr = LD(orbit["a_m"]), LD(orbit["L_m"]), LD(orbit["year_s"])
    pi = LD(4) * np.arctan(LD(1))
    delta = Lm / (2 * a)
    s3 = np.sqrt(LD(3))
    e = np.sqrt(1 + 2 * delta / s3 + 4 * delta * delta / 3) - 1
    inc = np.arctan(delta / (1 + delta / s3))
    for k in range(3):
        sigma = 2 * pi * k / 3
        M = 2 * pi * (t - LD(orbit.get("t_ref", 0.0))) / yr - sigma - LD(orbit.get("phase0", 0.0))
        psi = M + e * np.sin(M)
        xi, eta = a * (np.cos(psi) - e), a * np.sqrt(1 - e * e) * np.sin(psi)   # in the orbital plane
        x, y, z = xi * np.cos(inc), eta, xi * np.sin(inc)                       # tilt about y
        r[k, 0] = np.cos(sigma) * x - np.sin(sigma) * y                         # turn about z
        r[k, 1] = np.sin(sigma) * x + np.cos(sigma) * y
        r[k, 2] = z
    return r


def travel_times(orbit, r):
    if orbit["kind"] == "static":
        return [np.full(r.shape[2], LD(orbit["L_static"][i])) for i in range(6)]
    return [np.sqrt(np.sum((r[SR[l][1] - 1] - r[SR[l][0] - 1]) ** 2, axis=0)) / C for l in LINKS]


def second_path_links(hp, hc, lam, bet, orbit, t0, dt, order, margin):
    """Eq. 2.7-2.8 with readings A7, A11; one walker.  Returns y[6][N] long double."""
    N = hp.shape[0]
    t0, dt = LD(t0), LD(dt)
    t = t0 + np.arange(N).astype(LD) * dt
    lam, bet = LD(lam), LD(bet)
    k = np.array([-np.cos(bet) * np.cos(lam), -np.cos(bet) * np.sin(lam), -np.sin(bet)])
    v = np.array([-np.sin(bet) * np.cos(lam), -np.sin(bet) * np.sin(lam), np.cos(bet)])
    u = np.array([np.sin(lam), -np.cos(lam), LD(0)])
    r = positions(orbit, t)
    L = travel_times(orbit, r)
    hp, hc = hp.astype(LD), hc.astype(LD)
    y = np.zeros((6, N), dtype=LD)
    dot = lambda a, b: a[0] * b[0] + a[1] * b[1] + a[2] * b[2]
    for i, link in enumerate(LINKS):
        s, rc = SR[link]
        d = r[rc - 1] - r[s - 1]
        nh = d / np.sqrt(dot(d, d))
        un, vn, kn = dot(u, nh), dot(v, nh), dot(k, nh)
        xp, xc = un * un - vn * vn, un * vn
        ts = t - L[i] - dot(k, r[s - 1]) / C
        tr = t - dot(k, r[rc - 1]) / C
        dhp = neville_read(hp, t0, dt, order, t, ts) - neville_read(hp, t0, dt, order, t, tr)
        dhc = neville_read(hc, t0, dt, order, t, ts) - neville_read(hc, t0, dt, order, t, tr)
        y[i] = (xp * dhp + 2 * xc * dhc) / (2 * (1 - kn))
    y[:, :margin] = 0
    y[:, N - margin:] = 0
    return y


def second_path_tdi(y, orbit, t0, dt, order, generation, out_kind, mlo, mhi):
    """Eq. 2.9 / 2.10 (A9) with summed delays, all L at the output time (A10); Eq. 2.11."""
    N = y.shape[1]
    t0, dt = LD(t0), LD(dt)
    t = t0 + np.arange(N).astype(LD) * dt
    L = travel_times(orbit, positions(orbit, t))
    y = y.astype(LD)
    xyz = np.zeros((3, N), dtype=LD)
    for c in range(3):
        for sign, link, labels in load_terms(str(generation)):
            t_eval = t.copy()
            for lab in labels:
                t_eval = t_eval - L[lidx(cyc(lab, c))]
            ser = y[lidx(cyc(link, c))]
            val = ser if not labels else neville_read(ser, t0, dt, order, t, t_eval)
            xyz[c] += sign * val
    out = xyz
    if out_kind == 1:
        X, Y, Z = xyz
        out = np.stack([(Z - X) / np.sqrt(LD(2)), (X - 2 * Y + Z) / np.sqrt(LD(6)), (X + Y + Z) / np.sqrt(LD(3))])
    out[:, :mlo] = 0
    out[:, N - mhi:] = 0
    return out


def rel_l2(a, b):
    a, b = np.asarray(a, dtype=LD), np.asarray(b, dtype=LD)
    return float(np.sqrt(np.sum((a - b) ** 2) / np.sum(b ** 2)))


def _strain(rng, N, dt, t0):
    t = t0 + np.arange(N) * dt
    hp = sum(rng.standard_normal() * np.cos(2 * math.pi * f * t + rng.uniform(0, 6)) for f in rng.uniform(3e-4, 2e-2, 5))
    hc = sum(rng.standard_normal() * np.sin(2 * math.pi * f * t + rng.uniform(0, 6)) for f in rng.uniform(3e-4, 2e-2, 5))
    return 1e-20 * hp, 1e-20 * hc


@pytest.mark.parametrize("order", [3, 31])
@pytest.mark.parametrize("kind,N,t0,t_ref", [("static", 256, 0.0, 0.0), ("kepler1", 512, 0.0, 0.0),
                                             ("kepler1", 1024, 0.0, -7.0e6), ("kepler1", 512, 7.0e6, 0.0)])
def test_c12_second_path_agrees_with_the_oracle(orc, order, kind, N, t0, t_ref):
    rng = np.random.default_rng(N + order)
    dt, B = 5.0, 2
    orbit = synth.static_orbit() if kind == "static" else dict(synth.kepler_orbit(), t_ref=t_ref, phase0=0.4 if t_ref else 0.0)
    my = 24 if kind == "static" else 128
    mlo, mhi = my + 32, my + 16
    lam, bet = rng.uniform(0, 2 * math.pi, B), np.arcsin(rng.uniform(-0.9, 0.9, B))
    h = [_strain(rng, N, dt, t0) for _ in range(B)]
    hp, hc = np.stack([x[0] for x in h]), np.stack([x[1] for x in h])
    y_orc = orc.link_response(hp, hc, lam, bet, orbit, t0, dt, order, my)
    # at t0 = 7e6 s the second path's absolute times carry ulp(7e6 s) = 8e-13 s in long double, i.e. 1.5e-13
    # samples of delay error, amplified by 1/(1 - k.n) (the reason the oracle and the kernels work
    # relative to the sample index); the same orbital phase is reached at small times through t_ref
    tol = 2e-15 if t0 == 0.0 else 2e-12
    for b in range(B):
        y2 = second_path_links(hp[b], hc[b], lam[b], bet[b], orbit, t0, dt, order, my)
        for l in range(6):
            assert rel_l2(y_orc[b, l], y2[l]) < tol, (b, l, rel_l2(y_orc[b, l], y2[l]))
            assert np.all(y_orc[b, l, :my] == 0) and np.all(y_orc[b, l, N - my:] == 0)
        for gen in (15, 20):
            for out_kind in (0, 1):
                # both sides start from the SAME doubles (the oracle's links)
                ref = second_path_tdi(y_orc[b], orbit, t0, dt, order, gen, out_kind, mlo, mhi)
                got = orc.tdi(y_orc[b][None], orbit, t0, dt, order, gen, out_kind, mlo, mhi)[0]
                scale = max(float(np.sqrt(np.sum(ref[c] ** 2))) for c in range(3))
                for c in range(3):
                    err = float(np.sqrt(np.sum((got[c].astype(LD) - ref[c]) ** 2))) / scale
                    assert err < tol, (b, gen, out_kind, c, err)
                assert np.all(got[:, :mlo] == 0) and np.all(got[:, N - mhi:] == 0)


def test_second_path_would_notice_a_wrong_oracle(orc):
    """the check above is not vacuous: one order off, a shifted node window or a dropped TDI term
    move the second path by far more than 1e-15"""
    rng = np.random.default_rng(9)
    N, dt, order, my = 512, 5.0, 31, 128
    orbit = synth.kepler_orbit()
    hp, hc = rng.standard_normal((2, N))  # white: every tap matters
    y = second_path_links(hp, hc, 1.3, 0.4, orbit, 0.0, dt, order, my)
    y31 = orc.link_response(hp[None], hc[None], [1.3], [0.4], orbit, 0.0, dt, order, my)[0]
    assert rel_l2(y31[0], y[0]) < 2e-15
    y29 = orc.link_response(hp[None], hc[None], [1.3], [0.4], orbit, 0.0, dt, 29, my)[0]
    assert rel_l2(y29[0], y[0]) > 1e-3
    yo = orc.link_response(hp[None], hc[None], [1.3], [0.4], orbit, 0.0, dt, order, my)[0]
    t15 = second_path_tdi(yo, orbit, 0.0, dt, order, 15, 0, 160, 144)
    t20 = orc.tdi(yo[None], orbit, 0.0, dt, order, 20, 0, 160, 144)[0]
    assert rel_l2(t20[0], t15[0]) > 1e-3
