"""Pins of the oracle's S1 (modes -> polarisations), Eq. 2.1-2.6.

C7 of SURVEY.md section 8(c): closed-form l=2 harmonics, orthonormality by quadrature,
beta=0 twist, psi rotation, face-on closed form, and an independent numpy restatement of the
paper's single-sum formula Eq. 2.4-2.6 (with readings A3, A4) against the oracle's triple loop
of Eq. 2.1-2.3 (three separate Wigner-D matrices from factorial sums).
"""
import math

import numpy as np
import pytest

MODES = [(2, 2), (2, 1), (3, 3), (4, 4), (5, 5)]


# ---- closed forms -----------------------------------------------------------------------------
def test_swsh_l2_closed_forms(orc):
    rng = np.random.default_rng(1)
    for _ in range(20):
        iota, phi = rng.uniform(0, math.pi), rng.uniform(0, 2 * math.pi)
        c, s = math.cos(iota), math.sin(iota)
        ref = {
            2: math.sqrt(5 / (64 * math.pi)) * (1 + c) ** 2 * np.exp(2j * phi),
            -2: math.sqrt(5 / (64 * math.pi)) * (1 - c) ** 2 * np.exp(-2j * phi),
            1: math.sqrt(5 / (16 * math.pi)) * s * (1 + c) * np.exp(1j * phi),
            -1: math.sqrt(5 / (16 * math.pi)) * s * (1 - c) * np.exp(-1j * phi),
            0: math.sqrt(15 / (32 * math.pi)) * s * s,
        }
        for m, v in ref.items():
            assert abs(orc.swsh(2, m, iota, phi) - v) < 2e-16 * 4


def test_swsh_orthonormal_by_quadrature(orc):
    # int conj(Y_lm) Y_l'm' dOmega = delta_ll' delta_mm'; the phi integral is analytic (delta_mm'),
    # the iota integral is done by Gauss-Legendre in cos(iota) (integrand is a polynomial).
    x, w = np.polynomial.legendre.leggauss(24)
    iot = np.arccos(x)
    for m in range(-5, 6):
        ls = [l for l in range(2, 6) if l >= abs(m)]
        vals = {l: np.array([orc.swsh(l, m, i, 0.0).real for i in iot]) for l in ls}
        for l1 in ls:
            for l2 in ls:
                integral = 2 * math.pi * np.sum(w * vals[l1] * vals[l2])
                assert abs(integral - (1.0 if l1 == l2 else 0.0)) < 1e-13, (l1, l2, m)


def test_small_d_is_orthogonal_matrix(orc):
    for l in (2, 3, 5):
        beta = 0.7 + 0.1 * l
        d = np.array([[orc.wigner_small_d(l, mp, m, beta) for m in range(-l, l + 1)]
                      for mp in range(-l, l + 1)])
        assert np.max(np.abs(d @ d.T - np.eye(2 * l + 1))) < 1e-14


def _one_sample_inputs(rng, modes, B=3, N=4):
    M = len(modes)
    amp = rng.uniform(0.5, 2.0, size=(B, M, N))
    phase = rng.uniform(-50, 50, size=(B, M, N))
    iota = rng.uniform(0, math.pi, B)
    phi = rng.uniform(0, 2 * math.pi, B)
    psi = rng.uniform(0, math.pi, B)
    return amp, phase, iota, phi, psi


def test_face_on_22_closed_form(orc):
    rng = np.random.default_rng(2)
    amp, phase, _, phi, _ = _one_sample_inputs(rng, [(2, 2)])
    B = amp.shape[0]
    hp, hc = orc.modes_to_pol([2], [2], amp, phase, np.zeros(B), phi, np.zeros(B))
    A = math.sqrt(5 / (4 * math.pi))
    arg = phase[:, 0, :] - 2 * phi[:, None]
    assert np.max(np.abs(hp - A * amp[:, 0] * np.cos(arg))) < 1e-15 * 4
    assert np.max(np.abs(hc - A * amp[:, 0] * np.sin(arg))) < 1e-15 * 4


def test_psi_rotates_polarisations(orc):
    rng = np.random.default_rng(3)
    l, m = zip(*MODES)
    amp, phase, iota, phi, psi = _one_sample_inputs(rng, MODES)
    hp0, hc0 = orc.modes_to_pol(l, m, amp, phase, iota, phi, 0 * psi)
    hp, hc = orc.modes_to_pol(l, m, amp, phase, iota, phi, psi)
    c, s = np.cos(2 * psi)[:, None], np.sin(2 * psi)[:, None]
    assert np.max(np.abs(hp - (hp0 * c + hc0 * s))) < 1e-14
    assert np.max(np.abs(hc - (hc0 * c - hp0 * s))) < 1e-14


def test_beta_zero_twist_is_a_phase(orc):
    # beta = 0: h^J_lm = e^{i m (alpha+gamma)} h^CP_lm, i.e. phase_lm -> phase_lm - m (alpha+gamma)
    rng = np.random.default_rng(4)
    l, m = zip(*MODES)
    amp, phase, iota, phi, psi = _one_sample_inputs(rng, MODES)
    B, M, N = amp.shape
    alpha, gamma = rng.uniform(-3, 3, (B, N)), rng.uniform(-3, 3, (B, N))
    hp, hc = orc.modes_to_pol(l, m, amp, phase, iota, phi, psi, alpha, np.zeros((B, N)), gamma)
    ph2 = phase - np.array(m)[None, :, None] * (alpha + gamma)[:, None, :]
    hp2, hc2 = orc.modes_to_pol(l, m, amp, ph2, iota, phi, psi)
    assert np.max(np.abs(hp - hp2)) < 1e-13
    assert np.max(np.abs(hc - hc2)) < 1e-13


def test_linear_in_amplitude_and_zero(orc):
    rng = np.random.default_rng(5)
    l, m = zip(*MODES)
    amp, phase, iota, phi, psi = _one_sample_inputs(rng, MODES)
    B, M, N = amp.shape
    ang = [rng.uniform(0, 1, (B, N)) for _ in range(3)]
    hp, hc = orc.modes_to_pol(l, m, amp, phase, iota, phi, psi, *ang)
    hp3, hc3 = orc.modes_to_pol(l, m, 3 * amp, phase, iota, phi, psi, *ang)
    assert np.max(np.abs(hp3 - 3 * hp)) < 1e-13
    hz, hcz = orc.modes_to_pol(l, m, 0 * amp, phase, iota, phi, psi, *ang)
    assert np.all(hz == 0) and np.all(hcz == 0)


# ---- the paper's single-sum form, restated independently in numpy -------------------------------
def quat_pair(alpha, beta, gamma):
    """Eq. 2.5 with the 1/sqrt(2) normalisation (reading A3), as Qa = q0 + i q3, Qb = q2 + i q1."""
    q0 = np.cos(beta / 2) * np.cos((alpha + gamma) / 2)
    q1 = -np.sin(beta / 2) * np.sin((alpha - gamma) / 2)
    q2 = np.sin(beta / 2) * np.cos((alpha - gamma) / 2)
    q3 = np.cos(beta / 2) * np.sin((alpha + gamma) / 2)
    return q0 + 1j * q3, q2 + 1j * q1


def quat_mul(p, q):
    """Product of consecutive rotations R_p R_q in the (Qa, Qb) pair representation."""
    pa, pb = p
    qa, qb = q
    return pa * qa - np.conj(pb) * qb, pb * qa + np.conj(pa) * qb


def wigner_D_quat(l, mp, m, Qa, Qb):
    """Eq. 2.6 with reading A4 (second binomial C(l-m', l-rho-m); value = frakD^l_{m'm})."""
    pref = math.sqrt(math.factorial(l + m) * math.factorial(l - m)
                     / (math.factorial(l + mp) * math.factorial(l - mp)))
    A, Bq = abs(Qa) ** 2, abs(Qb) ** 2
    s = 0.0
    for rho in range(0, l + mp + 1):
        k2 = l - rho - m
        if k2 < 0 or k2 > l - mp:
            continue
        s += math.comb(l + mp, rho) * math.comb(l - mp, k2) * (-Bq / A) ** rho
    return pref * A ** (l - m) * Qa ** (mp + m) * Qb ** (m - mp) * s


def pol_single_sum(modes, amp, phase, angles, euler0, iota, phi, psi):
    """Eq. 2.4 for one sample."""
    q = quat_pair(*angles)
    if euler0 is not None:
        q = quat_mul(q, quat_pair(*euler0))
    q = quat_mul(q, quat_pair(phi, iota, 0.0))  # PAPER.md:74 footnote 1
    H = 0j
    for k, (l, m) in enumerate(modes):
        h = amp[k] * np.exp(-1j * phase[k])
        H += h * math.sqrt((2 * l + 1) / (4 * math.pi)) * wigner_D_quat(l, m, 2, *q)
        hm = (-1) ** l * np.conj(h)
        H += hm * math.sqrt((2 * l + 1) / (4 * math.pi)) * wigner_D_quat(l, -m, 2, *q)
    H *= np.exp(2j * psi)
    return H.real, -H.imag


@pytest.mark.parametrize("with_e0", [False, True])
def test_triple_loop_equals_single_sum(orc, with_e0):
    rng = np.random.default_rng(6)
    l, m = zip(*MODES)
    B, N = 4, 6
    amp, phase, iota, phi, psi = _one_sample_inputs(rng, MODES, B, N)
    alpha = rng.uniform(-6, 6, (B, N))
    beta = rng.uniform(0.05, 2.8, (B, N))
    gamma = rng.uniform(-6, 6, (B, N))
    e0 = rng.uniform(0.1, 1.5, (B, 3)) if with_e0 else None
    hp, hc = orc.modes_to_pol(l, m, amp, phase, iota, phi, psi, alpha, beta, gamma, euler0=e0)
    scale = np.sum(amp, axis=1)
    for b in range(B):
        for n in range(N):
            rp, rc = pol_single_sum(MODES, amp[b, :, n], phase[b, :, n],
                                    (alpha[b, n], beta[b, n], gamma[b, n]),
                                    None if e0 is None else e0[b], iota[b], phi[b], psi[b])
            assert abs(hp[b, n] - rp) < 1e-13 * scale[b, n]
            assert abs(hc[b, n] - rc) < 1e-13 * scale[b, n]


def test_aligned_equals_zero_angles(orc):
    rng = np.random.default_rng(7)
    l, m = zip(*MODES)
    amp, phase, iota, phi, psi = _one_sample_inputs(rng, MODES)
    B, M, N = amp.shape
    z = np.zeros((B, N))
    a = orc.modes_to_pol(l, m, amp, phase, iota, phi, psi)
    b = orc.modes_to_pol(l, m, amp, phase, iota, phi, psi, z, z, z)
    assert np.max(np.abs(a[0] - b[0])) < 1e-15 and np.max(np.abs(a[1] - b[1])) < 1e-15
