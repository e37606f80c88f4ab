"""GPU test of lisa_td_tdi2_static: S3 with its scratch (merged-stencil tables, fix-up list, range-check
words) in the library's file-scope device array instead of a stream-ordered temporary, for callers that
cannot call cudaMalloc (include/lisa_td.h).  Same kernels as lisa_td_tdi2 (Eq. 2.9-2.11),
so the output is compared with that existing path, on calls in a row that share the array: different
sizes, orbits, generations and orders, the earlier one leaving a non-empty fix-up list and tables of more
sample groups than the later one uses.

The file is named so that pytest collects it LAST; it must pass alone in a fresh process and after the
other tests."""
import math

import numpy as np
import pytest
import torch

from paper_2501_08261_b200 import synth

pytestmark = pytest.mark.gpu

TOL = 1e-13  # the bar of tests/test_gpu_tdi_anchors.py; the two paths run the same kernels, so 0 is expected


@pytest.fixture(scope="module")
def lib():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2501_08261_b200 import lib as L
    L.load()
    return L


def _both(lib, y, orbit, t0, dt, order, gen, out_kind, mlo, mhi, check=True):
    B, _, N = y.shape
    yd = torch.from_numpy(y).cuda()
    ref = torch.full((B, 3, N), float("nan"), dtype=torch.float64, device="cuda")
    got = torch.full((B, 3, N), float("nan"), dtype=torch.float64, device="cuda")
    lib.tdi2(B, N, t0, dt, order, gen, out_kind, mlo, mhi, yd, orbit, ref)          # existing path
    lib.check()
    lib.tdi2_static(B, N, t0, dt, order, gen, out_kind, mlo, mhi, yd, orbit, got, check=check)
    torch.cuda.synchronize()
    return ref.cpu().numpy(), got.cpu().numpy()


def _assert_same(ref, got, mlo, mhi):
    N = ref.shape[-1]
    assert np.all(np.isfinite(got))
    assert np.all(got[:, :, :mlo] == 0) and np.all(got[:, :, N - mhi:] == 0)
    scale = np.sqrt(np.mean(ref ** 2))
    assert scale > 0
    assert np.max(np.abs(got - ref)) <= TOL * scale


def test_static_scratch_matches_tdi2_on_calls_in_a_row(lib, orc):
    rng = np.random.default_rng(20250108)
    kep = synth.kepler_orbit()

    # call 1: 9000 samples (71 sample groups), 17 walkers, and a grid on which the delay L2 + L-2 crosses an
    # integer in the middle: the fix-up list is NOT empty and the range-check words are read (check = 1)
    B, N, order, t0 = 17, 9000, 31, 3.0e6
    L_mid = orc.orbit_eval(kep, t0 + 4500 * 5.5)[1]
    dt = float((L_mid[1] + L_mid[4]) / 3.0)
    D = [(orc.orbit_eval(kep, t0 + n * dt)[1][1] + orc.orbit_eval(kep, t0 + n * dt)[1][4]) / dt for n in (0, N - 1)]
    assert math.ceil(D[0]) != math.ceil(D[1]), "the crossing must fall inside the grid"
    mlo, mhi = int(math.ceil(7 * 8.5 / dt)) + 16, 16
    y = rng.standard_normal((B, 6, N))
    ref, got = _both(lib, y, kep, t0, dt, order, 20, 1, mlo, mhi)
    _assert_same(ref, got, mlo, mhi)

    # call 2, right behind it: fewer samples (20 groups: the other 51 tables of call 1 stay in the array),
    # no crossing (the list of call 1 must not be replayed), generation 1.5, X,Y,Z, enqueue-only (check = 0);
    # the device's free memory must not move across the call
    B2, N2, dt2, t02 = 5, 2500, 5.0, 9.0e6
    y2 = rng.standard_normal((B2, 6, N2))
    yd2 = torch.from_numpy(y2).cuda()
    ref2 = torch.empty((B2, 3, N2), dtype=torch.float64, device="cuda")
    got2 = torch.full((B2, 3, N2), float("nan"), dtype=torch.float64, device="cuda")
    lib.tdi2(B2, N2, t02, dt2, 31, 15, 0, 28, 16, yd2, kep, ref2)
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    lib.tdi2_static(B2, N2, t02, dt2, 31, 15, 0, 28, 16, yd2, kep, got2, check=False)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free_before, "lisa_td_tdi2_static took device memory"
    _assert_same(ref2.cpu().numpy(), got2.cpu().numpy(), 28, 16)

    # call 3: the paper's linear interpolation (other table geometry in the same array), odd N (cp.async path)
    B3, N3 = 3, 4097
    y3 = rng.standard_normal((B3, 6, N3))
    ref3, got3 = _both(lib, y3, kep, 5.0e6, 5.0, 1, 20, 1, 13, 2)
    _assert_same(ref3, got3, 13, 2)

    # call 4: an order without merged stencils (one thread per sample, no scratch), static arms
    ref4, got4 = _both(lib, y3, synth.static_orbit(), 0.0, 5.0, 7, 20, 1, 64, 8)
    _assert_same(ref4, got4, 64, 8)


def test_static_scratch_at_its_maximum_and_beyond(lib):
    rng = np.random.default_rng(7)
    kep = synth.kepler_orbit()
    N = lib.TDI2_STATIC_MAX_N
    y = rng.standard_normal((2, 6, N))
    ref, got = _both(lib, y, kep, 1.0e6, 5.0, 31, 20, 1, 28, 16)
    _assert_same(ref, got, 28, 16)
    # one sample more is rejected with a clear error before anything is launched
    yd = torch.zeros((1, 6, N + 2), dtype=torch.float64, device="cuda")
    out = torch.zeros((1, 3, N + 2), dtype=torch.float64, device="cuda")
    with pytest.raises(lib.LisaTdError) as e:
        lib.tdi2_static(1, N + 2, 1.0e6, 5.0, 31, 20, 1, 28, 16, yd, kep, out)
    assert "LISA_TD_TDI2_STATIC_MAX_N" in str(e.value) and str(N) in str(e.value)
    lib.check()
