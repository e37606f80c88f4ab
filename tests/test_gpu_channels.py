"""GPU parity of the TDI channel subsets of PAPER.md:362 (A, AE, AET): lisa_td_loglike_channels
against the oracle's Eq. 2.12-2.13 summed over the same channels (the oracle's sum over c with
the weights of the excluded channels set to zero, which IS that definition)."""
import numpy as np
import pytest
import torch

from paper_2501_08261_b200 import synth

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def lib():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2501_08261_b200 import lib as L
    L.load()
    return L


@pytest.mark.parametrize("N", [1 << 12, 1 << 9])  # the oracle FFT is radix 2
def test_channel_subsets_match_the_oracle(lib, orc, N):
    rng = np.random.default_rng(11)
    B, dt = 5, 5.0
    nf = N // 2 + 1
    tdi = rng.standard_normal((B, 3, N)) * np.array([1.0, 0.7, 1e-3])[None, :, None]
    data = rng.standard_normal((3, nf, 2))
    w = np.abs(rng.standard_normal((3, nf))) + 0.1
    kmin, kmax = 7, nf - 20
    plan = lib.Plan(B, N)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    got = {}
    for n_ch in (1, 2, 3):
        ll = torch.empty(B, dtype=torch.float64, device="cuda")
        dh = torch.empty_like(ll)
        hh = torch.empty_like(ll)
        # poison the excluded channels: they must not be read
        t = tdi.copy()
        t[:, n_ch:] = np.nan
        lib.loglike_channels(plan, B, N, n_ch, dev(t), dev(data), dev(w), kmin, kmax, ll, dh, hh)
        torch.cuda.synchronize()
        wm = w.copy()
        wm[n_ch:] = 0.0
        rll, rdh, rhh = orc.loglike(tdi, data, wm, kmin, kmax)
        for g, r in ((ll, rll), (dh, rdh), (hh, rhh)):
            g = g.cpu().numpy()
            assert np.all(np.isfinite(g))
            assert np.max(np.abs(g - r) / np.abs(r)) < 1e-9
        got[n_ch] = ll.cpu().numpy()
    ll3 = torch.empty(B, dtype=torch.float64, device="cuda")
    lib.loglike(plan, B, N, dev(tdi), dev(data), dev(w), kmin, kmax, ll3)
    torch.cuda.synchronize()
    assert np.array_equal(ll3.cpu().numpy(), got[3])  # n_channels = 3 is the plain call
    assert np.max(np.abs(got[1] - got[3])) > 0.0
    plan.close()


def test_bad_channel_count_is_rejected(lib):
    N = 1024
    plan = lib.Plan(1, N)
    z = torch.zeros((1, 3, N), dtype=torch.float64, device="cuda")
    d = torch.zeros((3, N // 2 + 1, 2), dtype=torch.float64, device="cuda")
    w = torch.zeros((3, N // 2 + 1), dtype=torch.float64, device="cuda")
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    for bad in (0, 4, -1):
        with pytest.raises(lib.LisaTdError):
            lib.loglike_channels(plan, 1, N, bad, z, d, w, 1, 100, out)
    plan.close()
