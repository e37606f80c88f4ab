"""Pin of the oracle's noise weights (orc_psd_weights; Eq. 2.14-2.15, readings
A14/A15/A17) that does NOT re-type Eq. 2.15.

The channel PSDs of Eq. 2.15 are what uncorrelated link-level noises become after TDI.  The oracle's
own TDI (orc_tdi, pinned by C2-C5 in test_oracle_response_tdi.py) gives the transfer of every noise
source into A, E, T on a static equal-arm constellation, so

    S_c(f) = S_op(f) * sum_{6 links} |T_{c,l}(f)|^2  +  S_acc(f) * sum_{6 test masses} |T_{c,tm}(f)|^2

with the standard couplings (the ones Eq. 2.15 was derived with):
  - optical-metrology noise: one independent stream per link, added to that y_{slr};
  - acceleration noise: one independent stream per test mass.  The test mass on spacecraft i that
    faces spacecraft j enters the link received at i from j at the reception time, a(t), and the
    link sent from i to j at the emission time, a(t - L), with the same sign.

`measured_sums` drives orc_tdi with unit monochromatic inputs, one source at a time, and sums the
squared responses.  The weights of the oracle are then compared with these sums: a wrong 8, 16 or 128,
a wrong (3 + 2 cos x + cos 2x), (2 + cos x), (1 - cos x) or sin^4(x/2), a missing arm length in the
argument (A14) or a wrong generation-2 factor each fail here.  Eq. 2.14's two shapes are pinned at
the frequencies the paper prints (their knees, where each bracket is exactly 2) and by their
power-law limits.
"""
import math

import numpy as np
import pytest

from paper_2501_08261_b200 import synth

LINKS = [1, 2, 3, -1, -2, -3]
SR = {1: (3, 2), 2: (1, 3), 3: (2, 1), -1: (2, 3), -2: (3, 1), -3: (1, 2)}  # link -> (sender, receiver)
LINK_OF = {sr: LINKS.index(l) for l, sr in SR.items()}                        # (s, r) -> link index 0..5
C = synth.C_LIGHT


def _responses(orc, gen, omega, phasors, L, dt):
    """phasors: [S][6] complex link amplitudes of S sources.  Returns T[S][3]: complex amplitude of
    A, E, T per source, from the oracle's TDI run on Re and Im of phasor * e^{i omega t}."""
    S = phasors.shape[0]
    N = 384
    orbit = dict(synth.static_orbit(), L_static=[L] * 6)
    t = np.arange(N) * dt
    e = np.exp(1j * omega * t)
    y = np.zeros((2 * S, 6, N))
    y[:S] = (phasors[:, :, None] * e).real
    y[S:] = (phasors[:, :, None] * e).imag
    mlo = int(math.ceil(7 * L / dt)) + 16
    out = orc.tdi(y, orbit, 0.0, dt, 31, gen, 1, mlo, 16)
    n = N // 2
    return (out[:S, :, n] + 1j * out[S:, :, n]) * np.exp(-1j * omega * t[n])


def measured_sums(orc, gen, f, L, dt=1.0):
    """(sum over links |T_c,l|^2, sum over test masses |T_c,tm|^2) for c = A, E, T at frequency f."""
    omega = 2 * math.pi * f
    oms = np.eye(6, dtype=complex)
    acc = np.zeros((6, 6), dtype=complex)
    k = 0
    for i in (1, 2, 3):
        for j in (1, 2, 3):
            if i == j:
                continue
            acc[k, LINK_OF[(j, i)]] += 1.0                           # received at i from j: a(t)
            acc[k, LINK_OF[(i, j)]] += np.exp(-1j * omega * L)       # sent from i to j: a(t - L)
            k += 1
    To = _responses(orc, gen, omega, oms, L, dt)
    Ta = _responses(orc, gen, omega, acc, L, dt)
    return np.sum(np.abs(To) ** 2, axis=0), np.sum(np.abs(Ta) ** 2, axis=0)


# bins of a (N = 10000, dt = 5 s) grid: df = 2e-5 Hz, so the knees the paper prints are bins
N_GRID, DT_GRID = 10000, 5.0
DF = 1.0 / (N_GRID * DT_GRID)


def _S(orc, acc, oms, L, gen):
    """channel PSDs S_A, S_E, S_T [nf] recovered from the oracle's weights, w = 4 df dt^2 / S (A17)"""
    w = orc.psd_weights(N_GRID, DT_GRID, acc, oms, L, gen)
    with np.errstate(divide="ignore"):
        return 4 * DF * DT_GRID ** 2 / w


@pytest.mark.parametrize("gen", [15, 20])
def test_eq_2_15_is_the_tdi_transfer_of_link_noises(orc, gen):
    L = synth.ARM / C                       # 8.339 s: x = 2 pi f L (reading A14)
    acc, oms = 3e-15, 15e-12
    S_acc_only = _S(orc, acc, 0.0, L, gen)
    S_oms_only = _S(orc, 0.0, oms, L, gen)
    S_both = _S(orc, acc, oms, L, gen)
    S15_oms = _S(orc, 0.0, oms, L, 15)
    # x = 2 pi f L from 0.005 to 3.7 rad (f up to 70 mHz on a dt = 1 s grid for the transfer)
    for k in (5, 20, 57, 100, 250, 400, 733, 1000, 1801, 2600, 3500):
        f = k * DF
        so, sa = measured_sums(orc, gen, f, L)
        # the responses come back as doubles of O(1) inputs: a sum of squares of size s is known to
        # ~2e-16 / sqrt(s) (T at low frequency is a 1e-8 remnant)
        tol = 1e-8 + 4e-15 / math.sqrt(min(so.min(), sa.min()))
        # the two noise kinds add (uncorrelated sources)
        assert np.allclose(S_both[:, k], S_acc_only[:, k] + S_oms_only[:, k], rtol=1e-13)
        # A and E are the same; T differs: ratios fix every trigonometric factor of Eq. 2.15
        assert abs(so[0] / so[1] - 1) < 1e-9 and abs(sa[0] / sa[1] - 1) < 1e-9
        assert abs(S_oms_only[2, k] / S_oms_only[0, k] / (so[2] / so[0]) - 1) < tol, (gen, k)
        assert abs(S_acc_only[2, k] / S_acc_only[0, k] / (sa[2] / sa[0]) - 1) < tol, (gen, k)
        assert S_oms_only[0, k] == S_oms_only[1, k] and S_acc_only[0, k] == S_acc_only[1, k]
        # absolute level: S_op and S_acc of Eq. 2.14 are common to the three channels, so
        # S_c / sum_c must be the SAME number for A and T, and equal to Eq. 2.14 at the printed knees
        s_op = S_oms_only[0, k] / so[0]
        s_acc = S_acc_only[0, k] / sa[0]
        assert abs(S_oms_only[2, k] / so[2] / s_op - 1) < tol
        assert abs(S_acc_only[2, k] / sa[2] / s_acc - 1) < tol
        # generation 2 = generation 1.5 x |1 - e^{-4 i omega L}|^2, measured, not typed (A14)
        if gen == 20:
            so15, _ = measured_sums(orc, 15, f, L)
            assert abs(S_oms_only[0, k] / S15_oms[0, k] / (so[0] / so15[0]) - 1) < tol


def test_eq_2_14_shapes_at_the_printed_knees(orc):
    """S_op and S_acc recovered from the weights through the measured TDI sums: the brackets of
    Eq. 2.14 equal 2 at their knees (0.4 mHz, 8 mHz, 2 mHz) and follow their
    power laws away from them; amplitudes enter squared (A15)."""
    L = synth.ARM / C
    acc, oms = 3e-15, 15e-12
    S_a = _S(orc, acc, 0.0, L, 15)
    S_o = _S(orc, 0.0, oms, L, 15)

    def s_op(k):
        return S_o[0, k] / measured_sums(orc, 15, k * DF, L)[0][0]

    def s_acc(k):
        return S_a[0, k] / measured_sums(orc, 15, k * DF, L)[1][0]

    def op_bracket(k):   # S_op / (o^2 (2 pi f / c)^2) = 1 + (2 mHz / f)^4
        return s_op(k) / (oms ** 2 * (2 * math.pi * k * DF / C) ** 2)

    def acc_bracket(k):  # S_acc (2 pi f)^4 / (a^2 (2 pi f / c)^2) = (1 + (0.4 mHz/f)^2)(1 + (f/8 mHz)^4)
        w = 2 * math.pi * k * DF
        return s_acc(k) * w ** 4 / (acc ** 2 * (w / C) ** 2)

    k2, k04, k8 = 100, 20, 400           # 2 mHz, 0.4 mHz, 8 mHz
    assert abs(op_bracket(k2) - 2.0) < 1e-7
    assert abs(op_bracket(2 * k2) - (1 + 1 / 16)) < 1e-7          # f^-4 above the knee
    assert abs(op_bracket(k2 // 2) - 17.0) < 1e-6                 # and below
    assert abs(acc_bracket(k04) - 2.0 * (1 + (1 / 20) ** 4)) < 1e-7
    assert abs(acc_bracket(k8) - 2.0 * (1 + (1 / 20) ** 2)) < 1e-7
    assert abs(acc_bracket(2 * k8) - 17.0 * (1 + (1 / 40) ** 2)) < 1e-6
    assert abs(acc_bracket(k04 // 2) - 5.0 * (1 + (1 / 40) ** 4)) < 1e-6
    # amplitudes enter squared
    assert np.allclose(_S(orc, 2 * acc, 0.0, L, 15)[:, 1:], 4 * S_a[:, 1:], rtol=1e-13)
    assert np.allclose(_S(orc, 0.0, 3 * oms, L, 15)[:, 1:], 9 * S_o[:, 1:], rtol=1e-13)


def test_generation_2_psd_zeros_and_dc(orc):
    """The generation-2 PSD vanishes at f = n / (4 L/c) (reading A16: the band must stay below the
    first one); on a grid that has a bin exactly there the weight blows up.  w = 0 at k = 0."""
    L, dt, N = 8.0, 4.0, 4096               # 1/(4L) = 1/32 Hz = bin N/8 of df = 1/(N dt)
    w20 = orc.psd_weights(N, dt, 3e-15, 15e-12, L, 20)
    w15 = orc.psd_weights(N, dt, 3e-15, 15e-12, L, 15)
    k0 = N // 8
    assert np.all(w20[:, 0] == 0) and np.all(w15[:, 0] == 0)
    for c in range(3):
        assert w20[c, k0] > 1e20 * w20[c, k0 - 7]               # sin(pi) in floating point
        assert 0.1 < w15[c, k0] / w15[c, k0 - 7] < 10           # generation 1.5 has no zero there
    # the first zero of the configs' arm (8.339 s) sits at 29.98 mHz, above the 20 mHz band edge
    assert 1.0 / (4 * synth.ARM / C) > 0.02
