"""Host-side checks of the C-ABI library that need no GPU: it loads, exports every symbol that
include/lisa_td.h declares, and rejects bad arguments before touching the device."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2501_08261_b200 import build, lib as L
    build.build()
    L.load()
    return L


def test_exports_every_declared_symbol(lib):
    hdr = open(os.path.join(ROOT, "include", "lisa_td.h")).read()
    declared = set(re.findall(r"LISA_TD_API[^;]*?\b(lisa_td_\w+)\s*\(", hdr))
    assert len(declared) >= 18
    assert declared == set(lib.EXPORTS)
    L = lib.load()
    for name in declared:
        assert hasattr(L, name), name


def test_version_and_error_string(lib):
    assert lib.version() >= 100
    assert isinstance(lib.last_error(), str)


def test_orbit_struct_layout_matches_header(lib):
    # int + pad, 5 doubles, 9 doubles, 6 doubles, one pointer, two ints (delay model, reading A22)
    assert C.sizeof(lib.Orbit) == 8 + 5 * 8 + 9 * 8 + 6 * 8 + 8 + 8
    assert lib.Orbit.tt_order.offset == 176 and lib.Orbit.tdi_nested.offset == 180


def test_argument_validation_happens_before_any_launch(lib):
    L = lib.load()
    orb = lib.make_orbit({"kind": "kepler1", "L_m": 2.5e9, "a_m": 1.495978707e11, "year_s": 365.25 * 86400})
    fake = C.c_void_p(0x1000)       # aligned, never dereferenced: validation fails first
    odd = C.c_void_p(0x1008)
    # bad order
    rc = L.lisa_td_link_response(1, 4096, 0.0, 5.0, 30, 128, fake, fake, fake, fake, C.byref(orb), fake, None)
    assert rc == -1 and "order" in lib.last_error()
    # B <= 0
    assert L.lisa_td_link_response(0, 4096, 0.0, 5.0, 31, 128, fake, fake, fake, fake, C.byref(orb), fake, None) == -1
    # NULL pointer
    assert L.lisa_td_link_response(1, 4096, 0.0, 5.0, 31, 128, None, fake, fake, fake, C.byref(orb), fake, None) == -1
    # misaligned pointer
    assert L.lisa_td_link_response(1, 4096, 0.0, 5.0, 31, 128, odd, fake, fake, fake, C.byref(orb), fake, None) == -2
    # margin too small for the orbit: |k.r|/c can reach ~500 s = 100 samples
    rc = L.lisa_td_link_response(1, 4096, 0.0, 5.0, 31, 64, fake, fake, fake, fake, C.byref(orb), fake, None)
    assert rc == -1 and "margin_y" in lib.last_error()
    # delay model flags outside {0, 1}
    bad = lib.make_orbit({"kind": "kepler1", "L_m": 2.5e9, "a_m": 1.495978707e11, "year_s": 365.25 * 86400,
                          "tt_order": 2})
    rc = L.lisa_td_tdi2(1, 4096, 0.0, 5.0, 31, 20, 1, 160, 144, fake, C.byref(bad), fake, None)
    assert rc == -1 and "tt_order" in lib.last_error()
    # TDI: bad generation, small margins
    assert L.lisa_td_tdi2(1, 4096, 0.0, 5.0, 31, 17, 1, 160, 144, fake, C.byref(orb), fake, None) == -1
    assert L.lisa_td_tdi2(1, 4096, 0.0, 5.0, 31, 20, 1, 20, 144, fake, C.byref(orb), fake, None) == -1
    assert L.lisa_td_tdi2(1, 4096, 0.0, 5.0, 31, 20, 1, 160, 4, fake, C.byref(orb), fake, None) == -1
    # modes: l out of range
    l = (C.c_int * 1)(9)
    m = (C.c_int * 1)(2)
    assert L.lisa_td_modes_to_pol(1, 16, 1, l, m, *([fake] * 11), None) == -1
    # loglike: band outside the spectrum, NULL plan
    assert L.lisa_td_loglike(None, 1, 16, fake, fake, fake, 0, 4, fake, None, None, None) == -1
    # workspace size helper
    assert L.lisa_td_response_tdi_workspace_bytes(2, 1024) >= 2 * 6 * 1024 * 8 + 8 * 12 * 3 * 44 * 8  # links + anchor tables (one per 128 samples)


def test_combined_calls_add_the_link_margin_to_the_tdi_margins(lib):
    """reading A7: TDI must not interpolate across the hard-zeroed edge of y.  lisa_td_response_tdi
    knows margin_y and rejects TDI margins that do not include it (lisa_td_tdi2 alone cannot know)."""
    L = lib.load()
    orb = lib.make_orbit({"kind": "kepler1", "L_m": 2.5e9, "a_m": 1.495978707e11, "year_s": 365.25 * 86400})
    fake = C.c_void_p(0x1000)
    args = lambda mlo, mhi: (1, 4096, 0.0, 5.0, 31, 128, 20, 1, mlo, mhi, fake, fake, fake, fake, C.byref(orb), fake, fake,
                             L.lisa_td_response_tdi_workspace_bytes(1, 4096), None)
    assert L.lisa_td_response_tdi(*args(30, 144)) == -1 and "margin_lo" in lib.last_error()
    assert L.lisa_td_response_tdi(*args(155, 144)) == -1 and "margin_y" in lib.last_error()
    assert L.lisa_td_response_tdi(*args(160, 143)) == -1 and "margin_hi" in lib.last_error()
    # the same TDI margins are fine for lisa_td_tdi2 on its own (validation passes; the NULL stream
    # launch is never reached here because there is no device: any other error is acceptable)
    rc = L.lisa_td_tdi2(1, 4096, 0.0, 5.0, 31, 20, 1, 30, 16, fake, C.byref(orb), fake, None)
    assert rc in (0, -4) or "margin" not in lib.last_error()


def test_probes_and_debug_switches_are_not_part_of_the_abi(lib):
    hdr = open(os.path.join(ROOT, "include", "lisa_td.h")).read()
    assert "probe" not in hdr and "debug" not in hdr
    L = lib.load()
    assert not hasattr(L, "lisa_td_probe_dfma") and not hasattr(L, "lisa_td_debug_force_generic")


def test_probe_library_exports_what_its_header_declares(lib):
    """the bench-only probe library (csrc/lisa_td_probe.h) loads without a GPU and exports every
    entry point its header declares; bench.py's roofline denominators come from these"""
    import re
    hdr = open(os.path.join(ROOT, "paper_2501_08261_b200", "csrc", "lisa_td_probe.h")).read()
    declared = sorted(set(re.findall(r"\b(lisa_td_probe_\w+)\s*\(", hdr)))
    assert declared == ["lisa_td_probe_dfma", "lisa_td_probe_fp64_operands", "lisa_td_probe_fp64_pipes"]
    P = lib._probe_lib()
    for name in declared:
        assert hasattr(P, name), name


def test_psd_weights_host_helper_matches_oracle(lib, orc):
    """the CUDA library's host helper against the oracle's (pinned in test_oracle_psd_transfer.py),
    EVERY bin, with a tolerance that follows the conditioning of Eq. 2.15: w ~ 1 / (sin^2 x sin^2 2x ...),
    so a rounding of x = 2 pi f L (the two sides form it in different precisions) moves w by
    2 |cot x| + 4 |cot 2x| relative per unit of x."""
    N, dt, arm = 4096, 5.0, 8.339
    k = np.arange(1, N // 2 + 1)
    x = 2 * np.pi * k / (N * dt) * arm
    for gen in (15, 20):
        a = lib.psd_weights(N, dt, 3e-15, 15e-12, arm, gen)
        b = orc.psd_weights(N, dt, 3e-15, 15e-12, arm, gen)
        assert np.all(a[:, 0] == 0) and np.all(b[:, 0] == 0)
        cond = 1 + x * (2 / np.abs(np.tan(x)) + 2 / np.abs(np.tan(x / 2)) + (4 / np.abs(np.tan(2 * x)) if gen == 20 else 0))
        rel = np.abs(a[:, 1:] - b[:, 1:]) / np.abs(b[:, 1:])
        assert np.all(rel <= 4e-15 * cond[None, :]), float(np.max(rel / cond[None, :]))
