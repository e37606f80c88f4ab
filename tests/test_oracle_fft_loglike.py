"""Pins of the oracle's S4 (FFT) and S5 (inner products / log-likelihood), C9 and C10 of SURVEY 8(c),
and of its noise-weight helper (Eq. 2.14-2.15 with readings A14, A15, A17)."""
import math

import numpy as np
import pytest

from paper_2501_08261_b200 import synth


def test_c9_fft_vs_naive_dft_numpy_and_parseval(orc):
    rng = np.random.default_rng(0)
    for N in (8, 64, 1024):
        x = rng.standard_normal(N)
        s = orc.fft_r2c(x)
        sc = np.sqrt(N) * 1.0
        assert np.max(np.abs(s - orc.dft_naive(x))) < 1e-15 * N  # the definition itself
        assert np.max(np.abs(s - np.fft.rfft(x))) < 1e-14 * sc * 4  # a library routine
        full = np.concatenate([s, np.conj(s[-2:0:-1])])
        assert abs(np.sum(np.abs(full) ** 2) / N - np.sum(x ** 2)) < 1e-12 * np.sum(x ** 2)
    # a pure tone lands in one bin with amplitude N/2
    N, k0 = 256, 19
    s = orc.fft_r2c(np.cos(2 * math.pi * k0 * np.arange(N) / N))
    assert abs(s[k0] - N / 2) < 1e-12 and np.max(np.abs(np.delete(s, k0))) < 1e-12


def test_fft_large_matches_numpy(orc):
    rng = np.random.default_rng(1)
    x = rng.standard_normal(1 << 16)
    s = orc.fft_r2c(x)
    ref = np.fft.rfft(x)
    assert np.linalg.norm(s - ref) / np.linalg.norm(ref) < 1e-15 * 8


def _setup(rng, N=512, B=3):
    nf = N // 2 + 1
    tdi = rng.standard_normal((B, 3, N))
    w = rng.uniform(0.5, 2.0, (3, nf))
    return tdi, w, nf


def test_c10_closed_forms(orc):
    rng = np.random.default_rng(2)
    N = 512
    tdi, w, nf = _setup(rng, N)
    kmin, kmax = 7, 200
    d = tdi[0]
    dspec = orc.spectrum3(d)  # [3][nf][2]
    D = dspec[..., 0] + 1j * dspec[..., 1]
    dd = np.sum(w[:, kmin:kmax + 1] * np.abs(D[:, kmin:kmax + 1]) ** 2)
    # log L(h = d) = (d|d)/2 ; log L(lambda d) = (lambda - lambda^2/2)(d|d) ; log L(0) = 0
    for lamb in (1.0, 0.3, -1.7, 0.0):
        ll, dh, hh = orc.loglike(lamb * d[None], dspec, w, kmin, kmax)
        assert abs(ll[0] - (lamb - lamb ** 2 / 2) * dd) < 1e-13 * dd
        assert abs(dh[0] - lamb * dd) < 1e-13 * dd and abs(hh[0] - lamb ** 2 * dd) < 1e-13 * dd
    # independent numpy evaluation of Eq. 2.12-2.13 on random templates (footnote 3 sign, A13)
    ll, dh, hh = orc.loglike(tdi, dspec, w, kmin, kmax)
    H = np.fft.rfft(tdi, axis=-1)
    sl = slice(kmin, kmax + 1)
    ref_dh = np.sum(w[None, :, sl] * (D[None, :, sl] * np.conj(H[:, :, sl])).real, axis=(1, 2))
    ref_hh = np.sum(w[None, :, sl] * np.abs(H[:, :, sl]) ** 2, axis=(1, 2))
    assert np.max(np.abs(dh - ref_dh)) < 1e-12 * dd and np.max(np.abs(hh - ref_hh)) < 1e-12 * dd
    assert np.max(np.abs(ll - (ref_dh - ref_hh / 2))) < 1e-12 * dd
    # footnote 3: log L + (d|d)/2 ... = -(h-d|h-d)/2
    diff = orc.loglike(tdi - d[None], dspec, w, kmin, kmax)[2]
    assert np.max(np.abs(ll - dd / 2 + diff / 2)) < 1e-12 * dd


def test_psd_weights_against_independent_form(orc):
    N, dt = 1 << 14, 5.0
    L = synth.ARM / synth.C_LIGHT
    w = orc.psd_weights(N, dt, 3e-15, 15e-12, L, 20)
    k = np.arange(1, N // 2 + 1)
    f = k / (N * dt)
    c = synth.C_LIGHT
    sacc = (3e-15) ** 2 * (1 + (4e-4 / f) ** 2) * (1 + (f / 8e-3) ** 4) / (2 * np.pi * f) ** 4 * (2 * np.pi * f / c) ** 2
    sop = (15e-12) ** 2 * (1 + (2e-3 / f) ** 4) * (2 * np.pi * f / c) ** 2
    x = 2 * np.pi * f * L
    sae = 8 * np.sin(x) ** 2 * (2 * sacc * (3 + 2 * np.cos(x) + np.cos(2 * x)) + sop * (2 + np.cos(x)))
    st = 16 * sop * (1 - np.cos(x)) * np.sin(x) ** 2 + 128 * sacc * np.sin(x) ** 2 * np.sin(x / 2) ** 4
    g = 4 * np.sin(2 * x) ** 2
    num = 4 * (1 / (N * dt)) * dt * dt
    band = (f > 1e-4) & (f < 0.02)
    assert np.max(np.abs(w[0, 1:][band] * sae[band] * g[band] / num - 1)) < 1e-11
    assert np.max(np.abs(w[2, 1:][band] * st[band] * g[band] / num - 1)) < 1e-11
    assert np.array_equal(w[0], w[1]) and np.all(w[:, 0] == 0)
    # generation 1.5 weights differ exactly by the factor 4 sin^2(2x)
    w15 = orc.psd_weights(N, dt, 3e-15, 15e-12, L, 15)
    assert np.max(np.abs(w15[0, 1:][band] / w[0, 1:][band] / g[band] - 1)) < 1e-12
    # low-frequency limit of S_T/S_AE ~ x^2-suppressed OMS term: T is the quiet channel
    assert w[2, 600] > w[0, 600]


def test_band_bins():
    assert synth.likelihood_band(1 << 20, 5.0) == (525, 104857)
