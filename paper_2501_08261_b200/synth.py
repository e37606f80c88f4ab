"""Seeded synthetic inputs for the five BASELINE.json configs.

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none
of the method's arithmetic (no response, TDI, interpolation, FFT or likelihood):
it only draws per-walker scalars from ``numpy.random.default_rng(seed)`` and fills
the input arrays -- mode amplitudes/phases, Euler angles, the laser-noise stream --
as closed-form functions of (scalars, sample index).  The arrays stand in for the
IMRPhenomT modes and NNLO angles of the paper's workload (a ~61-day MBHB at 5 s
cadence, Table I at PAPER.md:261-286), which need the waveform model
and are not available here.

Arrays are torch float64 tensors on ``device`` ('cpu' for the tests, 'cuda' for
full-size runs; the same bits are then copied to whichever side needs them).
"""
from __future__ import annotations

import math

import numpy as np
import torch

SEED0 = 250108261
T_SUN = 4.925490947e-6  # G Msun / c^3  [s]
C_LIGHT = 299792458.0
D_L = 6.1714e26  # 20 Gpc in metres (Table I scale)
TAU_MIN = 2000.0  # coalescence this long after the grid end [s]
MODES = [(2, 2), (2, 1), (3, 3), (4, 4), (5, 5)]
MODE_RATIO = {(2, 2): 1.0, (2, 1): 0.10, (3, 3): 0.40, (4, 4): 0.15, (5, 5): 0.05}
AU = 1.495978707e11
YEAR = 365.25 * 86400.0
ARM = 2.5e9

# margins (reading A7): y valid on [128, N-128), TDI on [160, N-144)
MARGIN_Y = 128
MARGIN_TDI_LO = 160
MARGIN_TDI_HI = 144

CONFIGS = {
    1: dict(name="tiny", N=1 << 12, B=1, modes=[(2, 2)], precessing=False, orbit="static"),
    2: dict(name="single_2month", N=1 << 20, B=1, modes=MODES, precessing=False, orbit="kepler1"),
    3: dict(name="precessing_batch", N=1 << 20, B=64, modes=MODES, precessing=True,
            orbit="kepler1"),
    4: dict(name="full_likelihood", N=1 << 20, B=256, modes=MODES, precessing=True,
            orbit="kepler1"),
    5: dict(name="stress", N=1 << 22, B=32, modes=MODES, precessing=True, orbit="kepler1"),
}


def static_orbit(L=ARM):
    r = []
    for k in range(3):
        th = 2.0 * math.pi * k / 3.0
        r.append([L / math.sqrt(3.0) * math.cos(th), L / math.sqrt(3.0) * 0.5 * math.sin(th),
                  L / math.sqrt(3.0) * (math.sqrt(3.0) / 2.0) * math.sin(th)])
    return {"kind": "static", "r_static": r, "L_static": [L / C_LIGHT] * 6}


def kepler_orbit(L=ARM):
    return {"kind": "kepler1", "L_m": L, "a_m": AU, "year_s": YEAR, "phase0": 0.0, "t_ref": 0.0}


def draw_scalars(config: int, B: int, seed: int | None = None) -> dict:
    """Per-walker scalars.  Walker b = centre * (1 + 1e-3 xi_b); walker 0 is the centre."""
    cfg = CONFIGS[config]
    rng = np.random.default_rng(SEED0 + config if seed is None else seed)
    c = {}
    if config == 1:
        c["Mc"] = rng.uniform(1e5, 1e6)
        c["M"] = c["Mc"] / 0.25 ** 0.6  # equal-mass total mass, only sets the angle scale
    else:
        M = 10.0 ** rng.uniform(5.0, 7.0)
        q = rng.uniform(1.0, 8.0)
        c["M"] = M
        c["Mc"] = M * (q / (1.0 + q) ** 2) ** 0.6
    c["tc_off"] = 0.0
    c["lam"] = rng.uniform(0.0, 2.0 * math.pi)
    c["beta_sky"] = math.asin(rng.uniform(-1.0, 1.0))
    c["psi"] = rng.uniform(0.0, math.pi)
    c["iota"] = math.acos(rng.uniform(-1.0, 1.0))
    c["phi"] = rng.uniform(0.0, 2.0 * math.pi)
    c["c_alpha"] = rng.uniform(0.1, 0.3)
    c["c_gamma"] = rng.uniform(0.1, 0.3)
    c["beta0"] = rng.uniform(0.0, 1.2)
    c["alpha0"] = rng.uniform(0.0, 2.0 * math.pi)
    c["gamma0"] = rng.uniform(0.0, 2.0 * math.pi)
    offs = rng.uniform(0.0, 2.0 * math.pi, size=len(MODES))
    xi = rng.standard_normal(size=(B, 11))
    xi[0] = 0.0
    out = {}
    names = ["M", "Mc", "tc_off", "lam", "beta_sky", "psi", "iota", "phi", "c_alpha", "c_gamma",
             "beta0"]
    for j, nm in enumerate(names):
        if nm == "tc_off":
            out[nm] = 1e-3 * TAU_MIN * xi[:, j]
        elif nm == "Mc":
            out[nm] = c["Mc"] * (1.0 + 1e-3 * xi[:, 0])  # Mc follows M
        else:
            out[nm] = c[nm] * (1.0 + 1e-3 * xi[:, j])
    out["alpha0"] = np.full(B, c["alpha0"])
    out["gamma0"] = np.full(B, c["gamma0"])
    out["mode_offset"] = {MODES[i]: float(offs[i]) for i in range(len(MODES))}
    out["mode_offset"][(2, 2)] = 0.0
    return out


def make_inputs(config: int, device="cpu", B: int | None = None, N: int | None = None,
                seed: int | None = None, dt: float = 5.0) -> dict:
    """Build the input set of one config.  B / N may be overridden for reduced test sizes."""
    cfg = CONFIGS[config]
    B = cfg["B"] if B is None else B
    N = cfg["N"] if N is None else N
    modes = cfg["modes"]
    M_ = len(modes)
    s = draw_scalars(config, B, seed)
    dev = torch.device(device)
    f64 = torch.float64
    n = torch.arange(N, dtype=f64, device=dev)
    t = n * dt
    amp = torch.empty((B, M_, N), dtype=f64, device=dev)
    phase = torch.empty((B, M_, N), dtype=f64, device=dev)
    alpha = beta = gamma = None
    if cfg["precessing"]:
        alpha = torch.empty((B, N), dtype=f64, device=dev)
        beta = torch.empty((B, N), dtype=f64, device=dev)
        gamma = torch.empty((B, N), dtype=f64, device=dev)
    for b in range(B):
        Mc = float(s["Mc"][b])
        tc = N * dt + TAU_MIN + float(s["tc_off"][b])
        theta = (tc - t) / (5.0 * T_SUN * Mc)
        ph22 = -2.0 * theta.pow(5.0 / 8.0)
        a22 = math.sqrt(4.0 * math.pi / 5.0) * (C_LIGHT * T_SUN * Mc / D_L) * theta.pow(-0.25)
        for k, (l, m) in enumerate(modes):
            phase[b, k] = (m / 2.0) * ph22 + s["mode_offset"][(l, m)]
            amp[b, k] = a22 * MODE_RATIO[(l, m)]
        if cfg["precessing"]:
            f22 = theta.pow(-3.0 / 8.0) / (8.0 * math.pi * T_SUN * Mc)
            inv_w = 1.0 / (math.pi * T_SUN * float(s["M"][b]) * f22)
            d = inv_w - inv_w[0]
            alpha[b] = float(s["alpha0"][b]) + float(s["c_alpha"][b]) * d
            gamma[b] = float(s["gamma0"][b]) - float(s["c_gamma"][b]) * d
            beta[b] = float(s["beta0"][b]) + 0.05 * (t / (N * dt))
    def vec(name):
        return torch.tensor(np.asarray(s[name], dtype=np.float64), dtype=f64, device=dev)
    out = dict(
        config=config, name=cfg["name"], B=B, N=N, dt=dt, t0=0.0, order=31,
        l=[lm[0] for lm in modes], m=[lm[1] for lm in modes],
        amp=amp, phase=phase, alpha=alpha, beta=beta, gamma=gamma,
        iota=vec("iota"), phi=vec("phi"), psi=vec("psi"),
        lam=vec("lam"), beta_sky=vec("beta_sky"),
        orbit=static_orbit() if cfg["orbit"] == "static" else kepler_orbit(),
        margin_y=MARGIN_Y, margin_lo=MARGIN_TDI_LO, margin_hi=MARGIN_TDI_HI,
        scalars=s,
    )
    return out


def laser_stream(N: int, seed: int = SEED0 + 5, scale: float = 1e-13) -> np.ndarray:
    """Config 5: white common laser-noise stream p[n] = scale * N(0,1) (reading A12)."""
    rng = np.random.default_rng(seed + 1000)
    return scale * rng.standard_normal(N)


def likelihood_band(N: int, dt: float, f_lo: float = 1e-4, f_hi: float = 0.02):
    """Inclusive bin range [kmin, kmax] of the inner-product band (reading A16)."""
    df = 1.0 / (N * dt)
    kmin = int(math.ceil(f_lo / df - 1e-9))
    kmax = int(math.floor(f_hi / df + 1e-9))
    return kmin, kmax


NOISE = dict(acc=3e-15, oms=15e-12, arm_s=ARM / C_LIGHT)  # config 4 amplitudes (A15)
