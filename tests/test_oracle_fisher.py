"""Pins of the oracle's Fisher matrix (oracle/lisa_oracle.c: orc_fisher; reading A19 of DESIGN.md,
PAPER.md:249).  None of them re-types the oracle's formula:

 - Parseval: with unit weights over the whole spectrum the frequency-domain inner product is a
   plain time-domain dot product, so for a model that is LINEAR in its parameters the Fisher
   matrix is the time-domain Gram matrix of the basis series (no FFT involved in the check).
 - the finite-difference step drops out exactly for a linear model; the matrix is symmetric and
   positive semi-definite.
 - Gamma = - Hessian of log L (Eq. 2.12 as read in A13) for a linear model, taken through the
   oracle's separately pinned log-likelihood with second differences.
"""
import numpy as np

N = 256


def _basis(rng, D):
    return rng.standard_normal((D, 3, N))


def _walkers(h0, basis, delta):
    D = basis.shape[0]
    out = np.empty((D + 1, 3, N))
    out[0] = h0
    for i in range(D):
        out[i + 1] = h0 + delta[i] * basis[i]
    return out


def test_linear_model_is_the_time_domain_gram_matrix(orc):
    """sum_{k=0}^{N/2} g_k Re(A_k conj B_k) = N sum_n a_n b_n / 1 with g = 1 at DC and Nyquist
    and 2 elsewhere (Parseval for real series)."""
    rng = np.random.default_rng(1)
    D = 4
    basis = _basis(rng, D)
    h0 = rng.standard_normal((3, N))
    delta = np.array([1e-3, 0.5, 2.0, 7e-2])
    w = np.full((3, N // 2 + 1), 2.0)
    w[:, 0] = 1.0
    w[:, -1] = 1.0
    w[1] *= 3.0   # per-channel weights must be honoured
    w[2] *= 0.25
    got = orc.fisher(_walkers(h0, basis, delta), delta, w, 0, N // 2)
    cw = np.array([1.0, 3.0, 0.25])
    want = N * np.einsum("icn,jcn,c->ij", basis, basis, cw)
    assert np.max(np.abs(got - want)) < 1e-12 * np.max(np.abs(want))


def test_step_independence_symmetry_and_psd(orc):
    rng = np.random.default_rng(2)
    D = 5
    basis = _basis(rng, D)
    h0 = rng.standard_normal((3, N))
    w = rng.uniform(0.5, 2.0, (3, N // 2 + 1))
    kmin, kmax = 7, 90
    d1 = np.array([1e-2, 3e-1, 1.0, 5.0, 2e-3])
    d2 = d1[::-1].copy()
    g1 = orc.fisher(_walkers(h0, basis, d1), d1, w, kmin, kmax)
    g2 = orc.fisher(_walkers(h0, basis, d2), d2, w, kmin, kmax)
    assert np.max(np.abs(g1 - g2)) < 1e-11 * np.max(np.abs(g1))
    assert np.max(np.abs(g1 - g1.T)) <= 1e-15 * np.max(np.abs(g1))
    assert np.min(np.linalg.eigvalsh(0.5 * (g1 + g1.T))) > -1e-12 * np.max(np.abs(g1))
    # the band matters: a different band gives a different matrix
    g3 = orc.fisher(_walkers(h0, basis, d1), d1, w, kmin, kmax - 20)
    assert np.max(np.abs(g3 - g1)) > 1e-3 * np.max(np.abs(g1))


def test_fisher_is_minus_the_hessian_of_loglike_for_a_linear_model(orc):
    """log L(theta) = (d|h) - (h|h)/2 with h linear in theta is exactly quadratic, so central
    second differences of orc_loglike give -Gamma with no truncation error."""
    rng = np.random.default_rng(3)
    D = 3
    basis = _basis(rng, D)
    h0 = rng.standard_normal((3, N))
    data = orc.spectrum3(rng.standard_normal((3, N)))
    w = rng.uniform(0.5, 2.0, (3, N // 2 + 1))
    kmin, kmax = 3, 100
    delta = np.array([0.3, 0.7, 1.1])
    gam = orc.fisher(_walkers(h0, basis, delta), delta, w, kmin, kmax)

    def ll(theta):
        h = h0 + np.einsum("i,icn->cn", theta, basis)
        return orc.loglike(h[None], data, w, kmin, kmax)[0][0]

    e = np.eye(D)
    for i in range(D):
        for j in range(D):
            s = 0.5
            hess = (ll(s * (e[i] + e[j])) - ll(s * (e[i] - e[j])) - ll(s * (e[j] - e[i])) + ll(-s * (e[i] + e[j]))) / (4 * s * s)
            assert abs(hess + gam[i, j]) < 1e-9 * np.max(np.abs(gam)), (i, j)
