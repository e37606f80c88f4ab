"""GPU parity: the CUDA path (through the C-ABI, via paper_2501_08261_b200.lib) against the
long-double CPU oracle on the same seeded inputs, stage by stage and end to end.

Tolerances: BASELINE.json north_star asks for rel-L2 <= 1e-11 per TDI
channel and 1e-9 relative on log L; h+/hx and the links are held to tighter bounds derived
from the fp64 arithmetic.  T of a heavy, low-frequency source on nearly equal arms is a ~1e-3
remnant of A/E, so its error is also measured against the common scale max(|A|,|E|,|T|).
"""
import math

import numpy as np
import pytest
import torch

from paper_2501_08261_b200 import synth

pytestmark = pytest.mark.gpu

TOL_TDI = 1e-11
TOL_LL = 1e-9


@pytest.fixture(scope="module")
def lib():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2501_08261_b200 import lib as L
    L.load()
    return L


def dev(a):
    return torch.as_tensor(np.ascontiguousarray(a, dtype=np.float64)).cuda()


def rel_l2(a, b):
    return float(np.linalg.norm(np.asarray(a) - np.asarray(b)) / np.linalg.norm(np.asarray(b)))


def gpu_s1(lib, l, m, amp, phase, iota, phi, psi, alpha=None, beta=None, gamma=None, euler0=None):
    B, M, N = amp.shape
    hp = torch.empty((B, N), dtype=torch.float64, device="cuda")
    hc = torch.empty_like(hp)
    d = lambda x: None if x is None else dev(x)
    lib.modes_to_pol(B, N, list(l), list(m), dev(amp), dev(phase), d(alpha), d(beta), d(gamma),
                     dev(iota), dev(phi), dev(psi), d(euler0), hp, hc)
    torch.cuda.synchronize()
    return hp.cpu().numpy(), hc.cpu().numpy()


def gpu_s2(lib, hp, hc, lam, bet, orbit, t0, dt, order, margin):
    B, N = hp.shape
    y = torch.full((B, 6, N), float("nan"), dtype=torch.float64, device="cuda")
    lib.link_response(B, N, t0, dt, order, margin, dev(hp), dev(hc), dev(lam), dev(bet), orbit, y)
    torch.cuda.synchronize()
    return y.cpu().numpy()


def gpu_s3(lib, y, orbit, t0, dt, order, gen, out_kind, mlo, mhi):
    B, _, N = y.shape
    out = torch.full((B, 3, N), float("nan"), dtype=torch.float64, device="cuda")
    lib.tdi2(B, N, t0, dt, order, gen, out_kind, mlo, mhi, dev(y), orbit, out)
    torch.cuda.synchronize()
    return out.cpu().numpy()


# ------------------------------------------------------------------------------------ S1
MODES5 = [(2, 2), (2, 1), (3, 3), (4, 4), (5, 5)]
MODES_GEN = [(2, 0), (3, 2), (4, 3), (5, 1), (6, 6), (7, 4), (8, 8), (8, 0), (3, 0), (6, 2)]


def _s1_inputs(rng, modes, B, N, big_phase=True):
    M = len(modes)
    amp = rng.uniform(0.5, 2.0, (B, M, N))
    phase = rng.uniform(-3e5, 3e5, (B, M, N)) if big_phase else rng.uniform(-50, 50, (B, M, N))
    iota, phi, psi = rng.uniform(0, math.pi, B), rng.uniform(0, 2 * math.pi, B), rng.uniform(0, math.pi, B)
    return amp, phase, iota, phi, psi


@pytest.mark.parametrize("modes", [[(2, 2)], MODES5, MODES_GEN])
@pytest.mark.parametrize("twisted", [False, True])
@pytest.mark.parametrize("with_e0", [False, True])
@pytest.mark.parametrize("force_generic", [0, 1, 2])
def test_s1_parity(lib, orc, modes, twisted, with_e0, force_generic):
    """force_generic=0 takes the five-mode TMA-pipelined kernel for the first two mode lists (N even),
    2 its load-everything-first variant, 1 the generic kernel."""
    if force_generic and len(modes) > 5:
        pytest.skip("already the generic kernel")
    rng = np.random.default_rng(11 + len(modes) + 2 * twisted + with_e0)
    B, N = 3, 2500  # several blocks / items and a ragged tail
    l, m = zip(*modes)
    amp, phase, iota, phi, psi = _s1_inputs(rng, modes, B, N)
    ang = [rng.uniform(-400, 400, (B, N)), rng.uniform(0, math.pi, (B, N)), rng.uniform(-400, 400, (B, N))] if twisted else [None] * 3
    e0 = rng.uniform(0.1, 1.5, (B, 3)) if with_e0 else None
    ref = orc.modes_to_pol(l, m, amp, phase, iota, phi, psi, *ang, euler0=e0)
    lib.debug_force_generic(force_generic)
    try:
        got = gpu_s1(lib, l, m, amp, phase, iota, phi, psi, *ang, euler0=e0)
    finally:
        lib.debug_force_generic(0)
    scale = np.sum(amp, axis=1)
    for g, r in zip(got, ref):
        # The bars of the first oracle commit, restored: max abs 5e-15 of the summed amplitudes (measured
        # 1.5e-15) and rel-L2 2e-15 for the paper's mode sets (measured 1.2e-15).  The ten-mode l <= 8 list
        # chains up to l+2 = 10 complex products per row over 2 n_modes rows: measured 3.0e-15, bar 5e-15.
        assert np.max(np.abs(g - r) / scale) < 5e-15
        assert rel_l2(g, r) < (2e-15 if len(modes) <= 5 else 5e-15)


@pytest.mark.parametrize("B,N", [(5, 1 << 16), (2, 1026), (3, 2501)])
def test_s1_five_mode_kernels_agree_bitwise(lib, B, N):
    """the TMA-pipelined persistent kernel (every block walks many (walker, tile) items when there are
    more than 296 of them; ragged last tile) against the load-everything-first kernel: same
    arithmetic, same bits; odd N takes the one-sample-per-thread variant in both modes"""
    rng = np.random.default_rng(N)
    l, m = zip(*MODES5)
    amp, phase, iota, phi, psi = _s1_inputs(rng, MODES5, B, N)
    ang = [rng.uniform(-400, 400, (B, N)), rng.uniform(0, math.pi, (B, N)), rng.uniform(-400, 400, (B, N))]
    outs = []
    for mode in (0, 2):
        lib.debug_force_generic(mode)
        try:
            outs.append(gpu_s1(lib, l, m, amp, phase, iota, phi, psi, *ang, euler0=None))
        finally:
            lib.debug_force_generic(0)
    assert np.array_equal(outs[0][0], outs[1][0]) and np.array_equal(outs[0][1], outs[1][1])
    assert np.all(np.isfinite(outs[0][0])) and np.abs(outs[0][0]).max() > 0.0


def test_s1_beta_pi(lib, orc):
    """A5: total beta = pi exactly (|Qa| = 0) must not divide by zero."""
    rng = np.random.default_rng(5)
    B, N = 2, 64
    l, m = zip(*MODES5)
    amp, phase, iota, phi, psi = _s1_inputs(rng, MODES5, B, N, big_phase=False)
    iota[:] = 0.0
    alpha, gamma = rng.uniform(-3, 3, (B, N)), rng.uniform(-3, 3, (B, N))
    beta = np.full((B, N), math.pi)
    ref = orc.modes_to_pol(l, m, amp, phase, iota, phi, psi, alpha, beta, gamma)
    got = gpu_s1(lib, l, m, amp, phase, iota, phi, psi, alpha, beta, gamma)
    for g, r in zip(got, ref):
        assert np.all(np.isfinite(g))
        assert np.max(np.abs(g - r)) < 2e-14


# ------------------------------------------------------------------------------------ S2
def _smooth_strain(rng, B, N, dt):
    t = np.arange(N) * dt
    hp, hc = np.zeros((B, N)), np.zeros((B, N))
    for b in range(B):
        for f in rng.uniform(2e-4, 2e-2, 6):
            hp[b] += rng.standard_normal() * np.cos(2 * math.pi * f * t + rng.uniform(0, 6.28))
            hc[b] += rng.standard_normal() * np.sin(2 * math.pi * f * t + rng.uniform(0, 6.28))
    return 1e-20 * hp, 1e-20 * hc


@pytest.mark.parametrize("order", [1, 5, 31, 63])
@pytest.mark.parametrize("orbit_kind", ["static", "kepler1"])
def test_s2_parity(lib, orc, order, orbit_kind):
    rng = np.random.default_rng(order + (7 if orbit_kind == "static" else 0))
    B, N, dt, margin, t0 = 2, 3000, 5.0, 160, 1.0e6
    hp, hc = _smooth_strain(rng, B, N, dt)
    lam, bet = rng.uniform(0, 2 * math.pi, B), np.arcsin(rng.uniform(-0.9, 0.9, B))
    orbit = synth.static_orbit() if orbit_kind == "static" else synth.kepler_orbit()
    ref = orc.link_response(hp, hc, lam, bet, orbit, t0, dt, order, margin)
    got = gpu_s2(lib, hp, hc, lam, bet, orbit, t0, dt, order, margin)
    assert np.all(got[:, :, :margin] == 0) and np.all(got[:, :, N - margin:] == 0)
    for b in range(B):
        for l in range(6):
            assert rel_l2(got[b, l], ref[b, l]) < 2e-13, (b, l)


@pytest.mark.parametrize("N,orbit_kind,tt_order", [(4097, "kepler1", 1), (4096, "kepler1", 0), (3001, "static", 0)])
def test_s2_linear_interpolation_kernel(lib, orc, orc_d, N, orbit_kind, tt_order):
    """order 1 (the paper's linear interpolation) has its own kernel: ragged walker
    groups (35 walkers = 32 + 3), odd N (scalar stores), first-order travel times"""
    rng = np.random.default_rng(N)
    B, dt, margin, t0 = 35, 5.0, 130, 2.0e6
    hp, hc = _smooth_strain(rng, B, N, dt)
    lam, bet = rng.uniform(0, 2 * math.pi, B), np.arcsin(rng.uniform(-0.9, 0.9, B))
    orbit = dict(synth.static_orbit() if orbit_kind == "static" else synth.kepler_orbit(), tt_order=tt_order)
    ref = orc.link_response(hp, hc, lam, bet, orbit, t0, dt, 1, margin)
    got = gpu_s2(lib, hp, hc, lam, bet, orbit, t0, dt, 1, margin)
    assert np.all(got[:, :, :margin] == 0) and np.all(got[:, :, N - margin:] == 0)
    lib.debug_force_generic(True)   # the staged kernel at H = 1 computes the same thing
    try:
        gen = gpu_s2(lib, hp, hc, lam, bet, orbit, t0, dt, 1, margin)
    finally:
        lib.debug_force_generic(False)
    ref_d = orc_d.link_response(hp, hc, lam, bet, orbit, t0, dt, 1, margin)
    errs = np.array([[rel_l2(got[b, l], ref[b, l]) for l in range(6)] for b in range(B)])
    errs_gen = np.array([[rel_l2(gen[b, l], ref[b, l]) for l in range(6)] for b in range(B)])
    floor = np.array([[rel_l2(ref_d[b, l], ref[b, l]) for l in range(6)] for b in range(B)])
    print("order 1: worst rel-L2 linear kernel", errs.max(), "staged kernel", errs_gen.max(), "oracle fp64 build", floor.max())
    # 210 series with random sky positions: some k fall near an arm, where y = dh / (2 (1 - k.n)) is a
    # difference of nearly equal reads; the bar is the usual 2e-13 or four times what the oracle's own
    # fp64 build loses on that series
    assert np.all(errs < np.maximum(2e-13, 4 * floor)), errs.max()
    assert np.all(errs_gen < np.maximum(2e-13, 4 * floor)), errs_gen.max()


def test_s2_generic_kernel_matches_specialised(lib, orc):
    rng = np.random.default_rng(3)
    B, N, dt, margin = 1, 2048, 5.0, 128
    hp, hc = _smooth_strain(rng, B, N, dt)
    lam, bet = rng.uniform(0, 6.28, B), np.arcsin(rng.uniform(-0.9, 0.9, B))
    orbit = synth.kepler_orbit()
    a = gpu_s2(lib, hp, hc, lam, bet, orbit, 0.0, dt, 31, margin)
    lib.debug_force_generic(True)
    try:
        b = gpu_s2(lib, hp, hc, lam, bet, orbit, 0.0, dt, 31, margin)
    finally:
        lib.debug_force_generic(False)
    assert rel_l2(a, b) < 1e-14  # two roundings of the same coefficients


# ------------------------------------------------------------------------------------ S3
@pytest.mark.parametrize("gen", [15, 20])
@pytest.mark.parametrize("out_kind", [0, 1])
@pytest.mark.parametrize("orbit_kind", ["static", "kepler1"])
@pytest.mark.parametrize("order,force_generic", [(31, False), (31, True), (1, False), (7, False)])
def test_s3_parity(lib, orc, gen, out_kind, orbit_kind, order, force_generic):
    rng = np.random.default_rng(gen + out_kind + order)
    B, N, dt, t0 = 11, 1000, 5.0, 3.0e6  # B > one walker chunk, N not a multiple of the tile
    mlo, mhi = 12 + (order + 1) // 2, (order + 1) // 2
    y = rng.standard_normal((B, 6, N))   # white: every tap matters
    orbit = synth.static_orbit() if orbit_kind == "static" else synth.kepler_orbit()
    ref = orc.tdi(y, orbit, t0, dt, order, gen, out_kind, mlo, mhi)
    lib.debug_force_generic(force_generic)
    try:
        got = gpu_s3(lib, y, orbit, t0, dt, order, gen, out_kind, mlo, mhi)
    finally:
        lib.debug_force_generic(False)
    assert np.all(got[:, :, :mlo] == 0) and np.all(got[:, :, N - mhi:] == 0)
    for b in range(B):
        for c in range(3):
            assert rel_l2(got[b, c], ref[b, c]) < 1e-13, (b, c)


@pytest.mark.parametrize("delays", [[3, 5, 4, 2, 6, 7], [1, 2, 2, 2, 1, 1]])
def test_s3_laser_noise_cancels_on_integer_delays(lib, delays):
    """C2 on the GPU: static integer-sample delays, three independent lasers -> X,Y,Z vanish.
    The first delay set runs the generic kernel, the second the merged-stencil kernel."""
    rng = np.random.default_rng(2)
    N, dt = 4096, 1.0
    orbit = {"kind": "static", "r_static": synth.static_orbit()["r_static"], "L_static": [float(d) for d in delays]}
    p = rng.standard_normal((3, N))
    S, R = [3, 1, 2, 2, 3, 1], [2, 3, 1, 3, 1, 2]
    y = np.zeros((1, 6, N))
    for l in range(6):
        d = delays[l]
        y[0, l, d:] = p[S[l] - 1, :N - d]
        y[0, l] -= p[R[l] - 1]
    mlo = 7 * max(delays) + 16
    for gen in (15, 20):
        out = gpu_s3(lib, y, orbit, 0.0, dt, 31, gen, 0, mlo, 16)
        assert np.max(np.abs(out[0, :, mlo + 64:N - 16])) < 1e-13 * np.sqrt(np.mean(y ** 2))


# ------------------------------------------------------------------------------------ chain
def _gpu_chain(lib, inp, gen=20, out_kind=1, want_y=False):
    B, N = inp["B"], inp["N"]
    d = lambda k: None if inp[k] is None else inp[k].cuda()
    hp = torch.empty((B, N), dtype=torch.float64, device="cuda")
    hc = torch.empty_like(hp)
    lib.modes_to_pol(B, N, inp["l"], inp["m"], d("amp"), d("phase"), d("alpha"), d("beta"), d("gamma"),
                     d("iota"), d("phi"), d("psi"), None, hp, hc)
    tdi = torch.empty((B, 3, N), dtype=torch.float64, device="cuda")
    ws = torch.empty(lib.response_tdi_workspace_bytes(B, N) // 8, dtype=torch.float64, device="cuda")
    lib.response_tdi(B, N, inp["t0"], inp["dt"], inp["order"], inp["margin_y"], gen, out_kind,
                     inp["margin_lo"], inp["margin_hi"], hp, hc, d("lam"), d("beta_sky"), inp["orbit"], tdi, ws)
    torch.cuda.synchronize()
    return hp.cpu().numpy(), hc.cpu().numpy(), ws[:B * 6 * N].view(B, 6, N).cpu().numpy(), tdi.cpu().numpy()


def _orc_chain(orc, inp, gen=20, out_kind=1, **kw):
    n = lambda k: None if inp[k] is None else inp[k].numpy()
    return orc.chain(inp["l"], inp["m"], n("amp"), n("phase"), n("iota"), n("phi"), n("psi"), n("lam"),
                     n("beta_sky"), inp["orbit"], inp["t0"], inp["dt"], inp["order"], inp["margin_y"], gen,
                     out_kind, inp["margin_lo"], inp["margin_hi"], alpha=n("alpha"), beta=n("beta"),
                     gamma=n("gamma"), **kw)


def _report(name, got, ref, rec=None, config=None, names="AET", floor_ref=None):
    """per-channel raw rel-L2 and error relative to the common scale of the three channels; floor_ref =
    the same series from the oracle's fp64 build (the rounding floor of any fp64 chain)"""
    common = max(np.linalg.norm(ref[c]) for c in range(3))
    raw = [rel_l2(got[c], ref[c]) for c in range(3)]
    com = [float(np.linalg.norm(got[c] - ref[c]) / common) for c in range(3)]
    flo = [None] * 3 if floor_ref is None else [rel_l2(floor_ref[c], ref[c]) for c in range(3)]
    print(f"{name}: raw {raw}  vs common scale {com}  fp64 floor {flo}")
    if rec is not None:
        for c in range(3):
            rec(config, name, names[c], raw=raw[c], common=com[c], floor=flo[c], tol=TOL_TDI,
                passed=raw[c] < TOL_TDI, note=None if raw[c] < TOL_TDI else "raw above the bar: see vs_common_scale and fp64_floor")
    return raw, com


@pytest.mark.parametrize("gen", [15, 20])
def test_config1_tiny(lib, orc, gen, parity_record):
    """configs[0]: N=2^12, (2,2) only, static equal arms, 1st + 2nd generation X,Y,Z."""
    inp = synth.make_inputs(1)
    ref = _orc_chain(orc, inp, gen, 0, want=("h", "y", "tdi"))
    hp, hc, y, tdi = _gpu_chain(lib, inp, gen, 0)
    assert rel_l2(hp, ref["hplus"]) < 2e-15 and rel_l2(hc, ref["hcross"]) < 2e-15
    for l in range(6):
        assert rel_l2(y[0, l], ref["y"][0, l]) < 2e-13
    raw, _ = _report(f"N=2^12 B=1 static arms generation {gen / 10:g} whole series", tdi[0], ref["tdi"][0], parity_record,
                     "configs[0]", "XYZ")
    assert max(raw) < TOL_TDI


@pytest.mark.parametrize("config,B,N", [(2, 1, 1 << 14), (3, 3, 1 << 14)])
def test_config23_reduced(lib, orc, orc_d, config, B, N, parity_record):
    """configs[1], [2] at reduced N (same generator, same cadence): 5 modes, Kepler orbits, A,E,T."""
    inp = synth.make_inputs(config, B=B, N=N)
    ref = _orc_chain(orc, inp, 20, 1, want=("h", "y", "tdi"))
    ref_d = _orc_chain(orc_d, inp, 20, 1, want=("tdi",))
    hp, hc, y, tdi = _gpu_chain(lib, inp, 20, 1)
    assert rel_l2(hp, ref["hplus"]) < 3e-15
    for b in range(B):
        for l in range(6):
            assert rel_l2(y[b, l], ref["y"][b, l]) < 2e-13
        raw, com = _report(f"reduced N=2^14 walker {b} whole series", tdi[b], ref["tdi"][b], parity_record,
                           f"configs[{config - 1}]", "AET", ref_d["tdi"][b])
        assert raw[0] < TOL_TDI and raw[1] < TOL_TDI
        assert com[2] < TOL_TDI          # T against the common scale
        assert raw[2] < 1e-8             # raw T: a ~1e-3 remnant on nearly equal arms


def test_loglike_parity(lib, orc, parity_record):
    """configs[3] at reduced size: FFT + inner products against the oracle's long-double FFT."""
    B, N = 4, 1 << 14
    inp = synth.make_inputs(4, B=B, N=N)
    dt = inp["dt"]
    kmin, kmax = synth.likelihood_band(N, dt)
    w = orc.psd_weights(N, dt, synth.NOISE["acc"], synth.NOISE["oms"], synth.NOISE["arm_s"], 20)
    ref = _orc_chain(orc, inp, 20, 1, want=("tdi",))
    data = orc.spectrum3(ref["tdi"][0])  # zero-noise injection = walker 0
    refll = _orc_chain(orc, inp, 20, 1, want=("loglike",), data_spec=data, weight=w, kmin=kmin, kmax=kmax)
    _, _, _, tdi = _gpu_chain(lib, inp, 20, 1)
    plan = lib.Plan(B, N)
    ll, dh, hh = (torch.empty(B, dtype=torch.float64, device="cuda") for _ in range(3))
    lib.loglike(plan, B, N, dev(tdi), dev(data), dev(w), kmin, kmax, ll, dh, hh)  # same weights, same data
    torch.cuda.synchronize()
    for got, key in ((ll, "loglike"), (dh, "dh"), (hh, "hh")):
        err = np.abs(got.cpu().numpy() - refll[key]) / np.abs(refll[key])
        print(key, err)
        parity_record("configs[3]", "reduced N=2^14 B=4, worst walker", key, raw=np.max(err), tol=TOL_LL, passed=np.max(err) < TOL_LL)
        assert np.max(err) < TOL_LL
    # closed form C10: log L(h = d) = (d|d)/2 for the injected walker
    assert abs(ll[0].item() - 0.5 * hh[0].item()) < 1e-9 * abs(hh[0].item())
    # spectrum entry point
    spec = torch.empty((B, 3, N // 2 + 1, 2), dtype=torch.float64, device="cuda")
    lib.spectrum(plan, B, N, dev(tdi), spec)
    torch.cuda.synchronize()
    s0 = spec[0].cpu().numpy()
    assert rel_l2(s0[:, kmin:kmax + 1], data[:, kmin:kmax + 1]) < 1e-10
    plan.close()


def test_laser_noise_suppression(lib, orc):
    """configs[4] / A12, P6: common laser noise at link level through TDI-2 on Kepler arms."""
    N, dt, order, margin = 1 << 14, 5.0, 31, 32
    orbit = synth.kepler_orbit()
    p = synth.laser_stream(N)
    yref = orc.laser_links(p, orbit, 0.0, dt, order, margin)
    y = torch.empty((6, N), dtype=torch.float64, device="cuda")
    lib.laser_links(N, 0.0, dt, order, margin, dev(p), orbit, y)
    torch.cuda.synchronize()
    yg = y.cpu().numpy()
    rms = np.sqrt(np.mean(yref ** 2))
    assert np.max(np.abs(yg - yref)) < 1e-11 * rms
    mlo, mhi = margin + 32, margin + 16
    ref = orc.tdi(yref[None], orbit, 0.0, dt, order, 20, 0, mlo, mhi)
    got = gpu_s3(lib, yg[None], orbit, 0.0, dt, order, 20, 0, mlo, mhi)
    assert np.max(np.abs(got - ref)) < 1e-11 * rms          # P6: absolute tolerance
    # suppression below 20 mHz (A12): windowed spectra of residual vs link noise
    win = np.kaiser(N, 30.0)
    f = np.fft.rfftfreq(N, dt)
    band = (f > 1e-3) & (f < 2e-2)
    X = np.abs(np.fft.rfft(win * got[0, 0]))[band]
    Y = np.abs(np.fft.rfft(win * yg[0]))[band]
    assert np.sqrt(np.mean(X ** 2) / np.mean(Y ** 2)) < 1e-5


def test_zero_strain_gives_zero(lib):
    B, N = 2, 4096
    z = np.zeros((B, N))
    y = gpu_s2(lib, z, z, np.array([1.0, 2.0]), np.array([0.3, -0.4]), synth.kepler_orbit(), 0.0, 5.0, 31, 128)
    assert np.all(y == 0)
    out = gpu_s3(lib, y, synth.kepler_orbit(), 0.0, 5.0, 31, 20, 1, 160, 144)
    assert np.all(out == 0)


def test_pipeline_host_matches_stagewise(lib, orc):
    """The end-to-end host call (chunked, two streams) equals the stage-by-stage device path."""
    B, N = 5, 1 << 13
    inp = synth.make_inputs(4, B=B, N=N)
    dt = inp["dt"]
    kmin, kmax = synth.likelihood_band(N, dt)
    w = lib.psd_weights(N, dt, synth.NOISE["acc"], synth.NOISE["oms"], synth.NOISE["arm_s"], 20)
    _, _, _, tdi = _gpu_chain(lib, inp, 20, 1)
    plan = lib.Plan(B, N)
    spec = torch.empty((B, 3, N // 2 + 1, 2), dtype=torch.float64, device="cuda")
    lib.spectrum(plan, B, N, dev(tdi), spec)
    data = spec[0].contiguous()
    ll = torch.empty(B, dtype=torch.float64, device="cuda")
    lib.loglike(plan, B, N, dev(tdi), data, dev(w), kmin, kmax, ll)
    torch.cuda.synchronize()
    pipe = lib.Pipeline(2, N, len(inp["l"]), True)   # chunk of 2 -> 3 chunks, last one ragged
    out = np.zeros(B)
    h = lambda k: inp[k].numpy()
    lib.pipeline_host(pipe, B, N, inp["l"], inp["m"], h("amp"), h("phase"), h("alpha"), h("beta"), h("gamma"),
                      h("iota"), h("phi"), h("psi"), h("lam"), h("beta_sky"), inp["t0"], dt, inp["order"],
                      inp["margin_y"], 20, inp["margin_lo"], inp["margin_hi"], inp["orbit"],
                      data.cpu().numpy(), w, kmin, kmax, out)
    assert np.max(np.abs(out - ll.cpu().numpy()) / np.abs(out)) < 1e-12
    # ... and the oracle's own chain, with its own injection (walker 0) and weights
    w_o = orc.psd_weights(N, dt, synth.NOISE["acc"], synth.NOISE["oms"], synth.NOISE["arm_s"], 20)
    data_o = orc.spectrum3(_orc_chain(orc, inp, 20, 1, want=("tdi",))["tdi"][0])
    ref = _orc_chain(orc, inp, 20, 1, want=("loglike",), data_spec=data_o, weight=w_o, kmin=kmin, kmax=kmax)
    out2 = np.zeros(B)
    lib.pipeline_host(pipe, B, N, inp["l"], inp["m"], h("amp"), h("phase"), h("alpha"), h("beta"), h("gamma"),
                      h("iota"), h("phi"), h("psi"), h("lam"), h("beta_sky"), inp["t0"], dt, inp["order"],
                      inp["margin_y"], 20, inp["margin_lo"], inp["margin_hi"], inp["orbit"], data_o, w_o, kmin, kmax, out2)
    assert np.max(np.abs(out2 - ref["loglike"]) / np.abs(ref["loglike"])) < TOL_LL
    pipe.close()
    plan.close()


def test_loglike_from_modes_is_the_stagewise_path_in_one_call(lib, orc):
    """lisa_td_loglike_from_modes (S1..S5 from device inputs, one call) against the four stage calls (bit for
    bit: the same kernels in the same order) and against the oracle's own chain."""
    B, N = 5, 1 << 13
    inp = synth.make_inputs(4, B=B, N=N)
    dt = inp["dt"]
    kmin, kmax = synth.likelihood_band(N, dt)
    w = orc.psd_weights(N, dt, synth.NOISE["acc"], synth.NOISE["oms"], synth.NOISE["arm_s"], 20)
    data = orc.spectrum3(_orc_chain(orc, inp, 20, 1, want=("tdi",))["tdi"][0])
    ref = _orc_chain(orc, inp, 20, 1, want=("loglike",), data_spec=data, weight=w, kmin=kmin, kmax=kmax)
    d = lambda k: None if inp[k] is None else inp[k].cuda()
    plan = lib.Plan(B, N)
    ws = torch.empty(lib.loglike_from_modes_workspace_bytes(B, N) // 8, dtype=torch.float64, device="cuda")
    ll, dh, hh = (torch.empty(B, dtype=torch.float64, device="cuda") for _ in range(3))
    lib.loglike_from_modes(plan, B, N, inp["l"], inp["m"], d("amp"), d("phase"), d("alpha"), d("beta"), d("gamma"),
                           d("iota"), d("phi"), d("psi"), d("lam"), d("beta_sky"), inp["t0"], dt, inp["order"],
                           inp["margin_y"], 20, inp["margin_lo"], inp["margin_hi"], inp["orbit"], dev(data), dev(w),
                           kmin, kmax, ll, dh, hh, ws)
    lib.check()
    for got, key in ((ll, "loglike"), (dh, "dh"), (hh, "hh")):
        assert np.max(np.abs(got.cpu().numpy() - ref[key]) / np.abs(ref[key])) < TOL_LL
    _, _, _, tdi = _gpu_chain(lib, inp, 20, 1)
    ll2 = torch.empty(B, dtype=torch.float64, device="cuda")
    lib.loglike(plan, B, N, dev(tdi), dev(data), dev(w), kmin, kmax, ll2)
    torch.cuda.synchronize()
    assert torch.equal(ll, ll2)
    # a workspace that is too small, or TDI margins that do not include margin_y, are rejected before any launch
    with pytest.raises(lib.LisaTdError):
        lib.loglike_from_modes(plan, B, N, inp["l"], inp["m"], d("amp"), d("phase"), d("alpha"), d("beta"), d("gamma"),
                               d("iota"), d("phi"), d("psi"), d("lam"), d("beta_sky"), inp["t0"], dt, inp["order"],
                               inp["margin_y"], 20, inp["margin_lo"], inp["margin_hi"], inp["orbit"], dev(data), dev(w),
                               kmin, kmax, ll, dh, hh, ws[:1000])
    with pytest.raises(lib.LisaTdError):
        lib.loglike_from_modes(plan, B, N, inp["l"], inp["m"], d("amp"), d("phase"), d("alpha"), d("beta"), d("gamma"),
                               d("iota"), d("phi"), d("psi"), d("lam"), d("beta_sky"), inp["t0"], dt, inp["order"],
                               inp["margin_y"], 20, 40, inp["margin_hi"], inp["orbit"], dev(data), dev(w),
                               kmin, kmax, ll, dh, hh, ws)
    plan.close()
