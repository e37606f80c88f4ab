"""GPU parity of the anchored merged-stencil TDI kernel (k3_tdi_mma) where its assumptions end.

The kernel evaluates the merged TDI stencils exactly at three anchor samples per group of 128 samples
(four 32-sample MMA tiles) and gives every row the quadratic through them; that is valid only while no
integer delay K = ceil(D) changes inside the group and the orbit is one smooth function over it.  Groups
where that fails are recomputed sample by sample (k3_tdi_fixup).  These tests put such tiles on purpose -- an integer delay crossing in the middle
of the grid, a tabulated orbit with a node every 80 samples -- and compare with the long-double
oracle on WHITE link series (every tap matters: a row served by the wrong window is wrong at O(1)).
Eq. 2.9-2.11; readings A10, A21, A22 of DESIGN.md.
"""
import math

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


def _gpu_tdi(lib, y, orbit, t0, dt, order, gen, out_kind, mlo, mhi):
    B, _, N = y.shape
    out = torch.full((B, 3, N), float("nan"), dtype=torch.float64, device="cuda")
    lib.tdi2(B, N, t0, dt, order, gen, out_kind, mlo, mhi, torch.from_numpy(y).cuda(), orbit, out)
    lib.check()
    return out.cpu().numpy()


def _assert_close(got, ref, mlo, mhi, tol=1e-13):
    N = ref.shape[-1]
    assert np.all(got[:, :, :mlo] == 0) and np.all(got[:, :, N - mhi:] == 0)
    for b in range(ref.shape[0]):
        for c in range(3):
            err = np.linalg.norm(got[b, c] - ref[b, c]) / np.linalg.norm(ref[b, c])
            assert err < tol, (b, c, err)
    # and row by row: one bad 32-sample tile must not hide in an L2 norm over thousands of samples
    scale = np.sqrt(np.mean(ref ** 2))
    assert np.max(np.abs(got - ref)) < 100 * tol * scale


@pytest.mark.parametrize("gen", [15, 20])
@pytest.mark.parametrize("nested", [0, 1])
def test_integer_delay_crossing_inside_a_tile(lib, orc, gen, nested):
    """dt is chosen so that the delay L2 + L-2 of Eq. 2.9's y_231 term equals exactly 3 samples in the
    middle of the grid: K = ceil(D) changes from one sample to the next inside a tile."""
    rng = np.random.default_rng(10 * gen + nested)
    B, N, order, t0 = 19, 2500, 31, 3.0e6
    orbit = dict(synth.kepler_orbit(), nested=nested, tt_order=nested)
    L_mid = orc.orbit_eval(orbit, t0 + 1237 * 5.5)[1]
    dt = float((L_mid[1] + L_mid[4]) / 3.0)            # links 2 and -2
    D = [(orc.orbit_eval(orbit, t0 + n * dt)[1][1] + orc.orbit_eval(orbit, t0 + n * dt)[1][4]) / dt for n in (0, N - 1)]
    assert math.ceil(D[0]) != math.ceil(D[1]), "the crossing must fall inside the grid"
    mlo, mhi = int(math.ceil(7 * 8.5 / dt)) + 16, 16
    y = rng.standard_normal((B, 6, N))
    for out_kind in (0, 1):
        ref = orc.tdi(y, orbit, t0, dt, order, gen, out_kind, mlo, mhi)
        got = _gpu_tdi(lib, y, orbit, t0, dt, order, gen, out_kind, mlo, mhi)
        _assert_close(got, ref, mlo, mhi)


@pytest.mark.parametrize("nested", [0, 1])
def test_table_orbit_with_a_node_every_80_samples(lib, orc, nested):
    """TABLE orbit (A21): every third tile straddles a table node, where the interpolant switches
    polynomial; those tiles must take the exact path, the others the anchors."""
    rng = np.random.default_rng(5 + nested)
    B, N, dt, order, t0, h, q = 5, 3000, 5.0, 31, 1.0e6, 400.0, 5
    kep = synth.kepler_orbit()
    n_tab = int(np.ceil(N * dt / h)) + 2 + 2 * q
    t_tab0 = t0 - q * h
    tab = np.stack([orc.orbit_eval(kep, t_tab0 + h * j)[0] for j in range(n_tab)])
    # a table that is NOT smooth from node to node (1e3 m of seeded jitter, 3e-6 s of light time), so
    # that the two polynomials around a node really differ
    tab = tab + 1e3 * rng.standard_normal(tab.shape)
    orbit = {"kind": "table", "r_tab": tab, "t_tab0": t_tab0, "dt_tab": h, "tab_order": q, "nested": nested,
             "tt_order": nested}
    mlo, mhi = 12 + 16, 16
    y = rng.standard_normal((B, 6, N))
    ref = orc.tdi(y, orbit, t0, dt, order, 20, 1, mlo, mhi)
    got = _gpu_tdi(lib, y, orbit, t0, dt, order, 20, 1, mlo, mhi)
    _assert_close(got, ref, mlo, mhi)


def test_anchored_rows_match_the_generic_kernel(lib):
    """same inputs through the one-thread-per-sample kernel (exact coefficients for every row) and the
    anchored kernel: the quadratic through three anchors reproduces every row to rounding"""
    rng = np.random.default_rng(1)
    B, N, dt, order, t0 = 33, 4000, 5.0, 31, 9.0e6
    orbit = synth.kepler_orbit()
    y = rng.standard_normal((B, 6, N))
    a = _gpu_tdi(lib, y, orbit, t0, dt, order, 20, 0, 28, 16)
    lib.debug_force_generic(1)
    try:
        b = _gpu_tdi(lib, y, orbit, t0, dt, order, 20, 0, 28, 16)
    finally:
        lib.debug_force_generic(0)
    assert np.max(np.abs(a - b)) < 2e-14 * np.sqrt(np.mean(b ** 2)) * 10


@pytest.mark.parametrize("N,B", [(70, 1), (130, 2), (257, 17), (1000, 16), (1153, 40), (6002, 40), (9000, 17)])
def test_short_and_ragged_grids(lib, orc, N, B):
    """fewer samples than one anchor group (128) or one MMA tile (32), odd N (cp.async path), grids that
    end inside a group, walker counts around the chunk size of 16; the two long grids give a persistent
    block more than one tile (148 blocks, 188 and 282 tiles), so the A fragments of the next tile are formed
    under the last -- ragged -- walker chunk of the current one"""
    rng = np.random.default_rng(N + B)
    dt, order, t0 = 5.0, 31, 5.0e6
    orbit = synth.kepler_orbit()
    mlo, mhi = 28, 16
    y = rng.standard_normal((B, 6, N))
    for gen in (15, 20):
        ref = orc.tdi(y, orbit, t0, dt, order, gen, 1, mlo, mhi)
        got = _gpu_tdi(lib, y, orbit, t0, dt, order, gen, 1, mlo, mhi)
        _assert_close(got, ref, mlo, mhi)
