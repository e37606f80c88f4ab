"""ctypes/numpy binding of the CPU oracle (oracle/lisa_oracle.c).

TEST INFRASTRUCTURE: importable only from tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs.  The product package
(paper_2501_08261_b200) never imports this module.

    orc = Oracle("ld")   # long-double truth
    orc = Oracle("d")    # plain fp64, the timed CPU baseline
"""
import ctypes as C

import numpy as np

from . import build as _build

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int)


class OrcOrbit(C.Structure):
    _fields_ = [
        ("kind", C.c_int),
        ("L_m", C.c_double),
        ("a_m", C.c_double),
        ("year_s", C.c_double),
        ("phase0", C.c_double),
        ("t_ref", C.c_double),
        ("r_static", (C.c_double * 3) * 3),
        ("L_static", C.c_double * 6),
        ("n_tab", C.c_int),
        ("tab_order", C.c_int),
        ("t_tab0", C.c_double),
        ("dt_tab", C.c_double),
        ("r_tab", C.POINTER(C.c_double)),
        ("tt_order", C.c_int),
        ("nested", C.c_int),
    ]


def make_orbit(d: dict) -> OrcOrbit:
    """d: {'kind': 'static'|'kepler1', ...} as produced by the input generators."""
    o = OrcOrbit()
    if d["kind"] == "static":
        o.kind = 0
        for i in range(3):
            for j in range(3):
                o.r_static[i][j] = float(d["r_static"][i][j])
        for k in range(6):
            o.L_static[k] = float(d["L_static"][k])
    elif d["kind"] == "kepler1":
        o.kind = 1
        o.L_m = float(d["L_m"])
        o.a_m = float(d["a_m"])
        o.year_s = float(d["year_s"])
        o.phase0 = float(d.get("phase0", 0.0))
        o.t_ref = float(d.get("t_ref", 0.0))
    elif d["kind"] == "table":
        o.kind = 2
        tab = np.ascontiguousarray(d["r_tab"], dtype=np.float64)
        assert tab.ndim == 3 and tab.shape[1:] == (3, 3)
        o._keep = tab  # keep the array alive as long as the struct
        o.n_tab, o.tab_order = tab.shape[0], int(d.get("tab_order", 7))
        assert o.tab_order % 2 == 1 and o.n_tab > o.tab_order
        o.t_tab0, o.dt_tab = float(d["t_tab0"]), float(d["dt_tab"])
        o.r_tab = tab.ctypes.data_as(C.POINTER(C.c_double))
    else:
        raise ValueError(d["kind"])
    o.tt_order = int(d.get("tt_order", 0))  # reading A22
    o.nested = int(d.get("nested", 0))
    return o


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _p(a):
    return None if a is None else a.ctypes.data_as(_dp)


class Oracle:
    def __init__(self, real: str = "ld"):
        libs = _build.build()
        self.real = real
        self.lib = C.CDLL(libs[real])
        L = self.lib
        L.orc_sizeof_real.restype = C.c_int
        L.orc_num_threads.restype = C.c_int
        L.orc_delay_read.restype = C.c_double
        L.orc_delay_read.argtypes = [_dp, C.c_long, C.c_long, C.c_double, C.c_int]
        L.orc_lagrange_coeffs.argtypes = [C.c_int, C.c_double, _dp]
        L.orc_wigner_small_d.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, _dp]
        L.orc_swsh.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, _dp, _dp]
        L.orc_orbit_eval.argtypes = [C.POINTER(OrcOrbit), C.c_double, _dp, _dp]
        L.orc_orbit_state.argtypes = [C.POINTER(OrcOrbit), C.c_double, _dp, _dp]
        L.orc_nested_delay.restype = C.c_double
        L.orc_nested_delay.argtypes = [C.POINTER(OrcOrbit), C.c_double, _ip, C.c_int]
        L.orc_laser_links3.argtypes = [C.c_long, C.c_double, C.c_double, C.c_int, C.c_long, _dp,
                                       C.POINTER(OrcOrbit), _dp]
        L.orc_modes_to_pol.argtypes = [C.c_int, C.c_long, C.c_int, _ip, _ip] + [_dp] * 9 + [
            C.c_long, C.c_long, _dp, _dp]
        L.orc_link_response.argtypes = [C.c_int, C.c_long, C.c_double, C.c_double, C.c_int,
                                        C.c_long, _dp, _dp, _dp, _dp, C.POINTER(OrcOrbit),
                                        C.c_long, C.c_long, _dp]
        L.orc_laser_links.argtypes = [C.c_long, C.c_double, C.c_double, C.c_int, C.c_long, _dp,
                                      C.POINTER(OrcOrbit), _dp]
        L.orc_tdi.argtypes = [C.c_int, C.c_long, C.c_double, C.c_double, C.c_int, C.c_int, C.c_int,
                              C.c_long, C.c_long, _dp, C.POINTER(OrcOrbit), C.c_long, C.c_long, _dp]
        L.orc_fft_r2c.argtypes = [C.c_long, _dp, _dp]
        L.orc_dft_naive.argtypes = [C.c_long, _dp, _dp]
        L.orc_spectrum3.argtypes = [C.c_long, _dp, _dp]
        L.orc_loglike.argtypes = [C.c_int, C.c_long, _dp, _dp, _dp, C.c_long, C.c_long, _dp, _dp,
                                  _dp]
        L.orc_upsample2.argtypes = [C.c_int, C.c_long, _dp, _dp]
        L.orc_fisher.argtypes = [C.c_int, C.c_long, _dp, _dp, _dp, C.c_long, C.c_long, _dp]
        L.orc_psd_weights.argtypes = [C.c_long, C.c_double, C.c_double, C.c_double, C.c_double,
                                      C.c_int, _dp]
        L.orc_chain.argtypes = (
            [C.c_int, C.c_long, C.c_int, _ip, _ip] + [_dp] * 9
            + [C.c_double, C.c_double, C.c_int, _dp, _dp, C.POINTER(OrcOrbit), C.c_long, C.c_int,
               C.c_int, C.c_long, C.c_long, C.c_long, C.c_long]
            + [_dp] * 4 + [_dp, _dp, C.c_long, C.c_long, _dp, _dp, _dp])

    # -- small pieces -------------------------------------------------------
    def sizeof_real(self):
        return self.lib.orc_sizeof_real()

    def num_threads(self):
        return self.lib.orc_num_threads()

    def lagrange_coeffs(self, order, eps):
        c = np.zeros(order + 1)
        self.lib.orc_lagrange_coeffs(order, float(eps), _p(c))
        return c

    def delay_read(self, x, n, D, order):
        x = _f64(x)
        return self.lib.orc_delay_read(_p(x), x.size, int(n), float(D), int(order))

    def wigner_small_d(self, l, mp, m, beta):
        out = C.c_double()
        self.lib.orc_wigner_small_d(l, mp, m, float(beta), C.byref(out))
        return out.value

    def swsh(self, l, m, iota, phi):
        re, im = C.c_double(), C.c_double()
        self.lib.orc_swsh(l, m, float(iota), float(phi), C.byref(re), C.byref(im))
        return complex(re.value, im.value)

    def orbit_eval(self, orbit, t):
        o = make_orbit(orbit)
        r = np.zeros(9)
        L = np.zeros(6)
        self.lib.orc_orbit_eval(C.byref(o), float(t), _p(r), _p(L))
        return r.reshape(3, 3), L

    def orbit_state(self, orbit, t):
        o = make_orbit(orbit)
        r = np.zeros(9)
        v = np.zeros(9)
        self.lib.orc_orbit_state(C.byref(o), float(t), _p(r), _p(v))
        return r.reshape(3, 3), v.reshape(3, 3)

    def nested_delay(self, orbit, t, labels):
        o = make_orbit(orbit)
        lab = np.ascontiguousarray(labels, dtype=np.int32)
        return self.lib.orc_nested_delay(C.byref(o), float(t), lab.ctypes.data_as(_ip), lab.size)

    # -- stages -------------------------------------------------------------
    @staticmethod
    def _modes(l, m):
        la = np.ascontiguousarray(l, dtype=np.int32)
        ma = np.ascontiguousarray(m, dtype=np.int32)
        return la, ma, la.ctypes.data_as(_ip), ma.ctypes.data_as(_ip)

    def modes_to_pol(self, l, m, amp, phase, iota, phi, psi, alpha=None, beta=None, gamma=None,
                     euler0=None, n_lo=0, n_hi=None):
        amp, phase = _f64(amp), _f64(phase)
        B, M, N = amp.shape
        n_hi = N if n_hi is None else n_hi
        la, ma, lp, mp = self._modes(l, m)
        assert la.size == M
        ang = [None if a is None else _f64(a) for a in (alpha, beta, gamma)]
        e0 = None if euler0 is None else _f64(euler0)
        iota, phi, psi = _f64(iota), _f64(phi), _f64(psi)
        hp, hc = np.zeros((B, N)), np.zeros((B, N))
        rc = self.lib.orc_modes_to_pol(B, N, M, lp, mp, _p(amp), _p(phase), _p(ang[0]), _p(ang[1]),
                                       _p(ang[2]), _p(iota), _p(phi), _p(psi), _p(e0), n_lo, n_hi,
                                       _p(hp), _p(hc))
        assert rc == 0, rc
        return hp, hc

    def link_response(self, hplus, hcross, lam, beta_sky, orbit, t0, dt, order, margin, n_lo=0,
                      n_hi=None):
        hplus, hcross = _f64(hplus), _f64(hcross)
        B, N = hplus.shape
        n_hi = N if n_hi is None else n_hi
        lam, beta_sky = _f64(lam), _f64(beta_sky)
        o = make_orbit(orbit)
        y = np.zeros((B, 6, N))
        rc = self.lib.orc_link_response(B, N, t0, dt, order, margin, _p(hplus), _p(hcross), _p(lam),
                                        _p(beta_sky), C.byref(o), n_lo, n_hi, _p(y))
        assert rc == 0, rc
        return y

    def laser_links(self, p, orbit, t0, dt, order, margin):
        p = _f64(p)
        o = make_orbit(orbit)
        y = np.zeros((6, p.size))
        rc = self.lib.orc_laser_links(p.size, t0, dt, order, margin, _p(p), C.byref(o), _p(y))
        assert rc == 0, rc
        return y

    def laser_links3(self, p3, orbit, t0, dt, order, margin):
        p3 = _f64(p3)
        assert p3.ndim == 2 and p3.shape[0] == 3
        o = make_orbit(orbit)
        y = np.zeros((6, p3.shape[1]))
        rc = self.lib.orc_laser_links3(p3.shape[1], t0, dt, order, margin, _p(p3), C.byref(o), _p(y))
        assert rc == 0, rc
        return y

    def tdi(self, y, orbit, t0, dt, order, generation, out_kind, margin_lo, margin_hi, n_lo=0,
            n_hi=None):
        y = _f64(y)
        B, six, N = y.shape
        assert six == 6
        n_hi = N if n_hi is None else n_hi
        o = make_orbit(orbit)
        out = np.zeros((B, 3, N))
        rc = self.lib.orc_tdi(B, N, t0, dt, order, generation, out_kind, margin_lo, margin_hi,
                              _p(y), C.byref(o), n_lo, n_hi, _p(out))
        assert rc == 0, rc
        return out

    def fft_r2c(self, x):
        x = _f64(x)
        s = np.zeros((x.size // 2 + 1, 2))
        rc = self.lib.orc_fft_r2c(x.size, _p(x), _p(s))
        assert rc == 0, rc
        return s[:, 0] + 1j * s[:, 1]

    def dft_naive(self, x):
        x = _f64(x)
        s = np.zeros((x.size // 2 + 1, 2))
        self.lib.orc_dft_naive(x.size, _p(x), _p(s))
        return s[:, 0] + 1j * s[:, 1]

    def spectrum3(self, tdi):
        """[3][N] -> float64 [3][N/2+1][2]"""
        tdi = _f64(tdi)
        N = tdi.shape[-1]
        s = np.zeros((3, N // 2 + 1, 2))
        rc = self.lib.orc_spectrum3(N, _p(tdi), _p(s))
        assert rc == 0, rc
        return s

    def loglike(self, tdi, data_spec, weight, kmin, kmax):
        tdi, data_spec, weight = _f64(tdi), _f64(data_spec), _f64(weight)
        B, three, N = tdi.shape
        ll, dh, hh = np.zeros(B), np.zeros(B), np.zeros(B)
        rc = self.lib.orc_loglike(B, N, _p(tdi), _p(data_spec), _p(weight), kmin, kmax, _p(ll),
                                  _p(dh), _p(hh))
        assert rc == 0, rc
        return ll, dh, hh

    def upsample2(self, coarse):
        """[B][N/2+1] on the 2 dt grid -> [B][N] on the dt grid (linear interpolation)"""
        coarse = _f64(coarse)
        B, Nc = coarse.shape
        N = 2 * (Nc - 1)
        out = np.zeros((B, N))
        rc = self.lib.orc_upsample2(B, N, _p(coarse), _p(out))
        assert rc == 0, rc
        return out

    def fisher(self, tdi, delta, weight, kmin, kmax):
        """tdi: [D+1][3][N] (walker 0 = centre, walker i = theta + delta_i e_i) -> [D][D]"""
        tdi, delta, weight = _f64(tdi), _f64(delta), _f64(weight)
        D = tdi.shape[0] - 1
        N = tdi.shape[-1]
        out = np.zeros((D, D))
        rc = self.lib.orc_fisher(D, N, _p(tdi), _p(delta), _p(weight), kmin, kmax, _p(out))
        assert rc == 0, rc
        return out

    def psd_weights(self, N, dt, acc_noise, oms_noise, arm_s, generation):
        w = np.zeros((3, N // 2 + 1))
        self.lib.orc_psd_weights(N, dt, acc_noise, oms_noise, arm_s, generation, _p(w))
        return w

    def chain(self, l, m, amp, phase, iota, phi, psi, lam, beta_sky, orbit, t0, dt, order,
              margin_y, generation, out_kind, margin_lo, margin_hi, alpha=None, beta=None,
              gamma=None, euler0=None, n_lo=0, n_hi=None, want=("tdi",), data_spec=None,
              weight=None, kmin=0, kmax=0):
        """Full chain in REAL.  want: subset of {'h','y','tdi','loglike'} -> dict."""
        amp, phase = _f64(amp), _f64(phase)
        B, M, N = amp.shape
        n_hi = N if n_hi is None else n_hi
        la, ma, lp, mp = self._modes(l, m)
        ang = [None if a is None else _f64(a) for a in (alpha, beta, gamma)]
        e0 = None if euler0 is None else _f64(euler0)
        iota, phi, psi, lam, beta_sky = map(_f64, (iota, phi, psi, lam, beta_sky))
        o = make_orbit(orbit)
        hp = np.zeros((B, N)) if "h" in want else None
        hc = np.zeros((B, N)) if "h" in want else None
        y = np.zeros((B, 6, N)) if "y" in want else None
        tdi = np.zeros((B, 3, N)) if "tdi" in want else None
        ll = dh = hh = None
        ds = w = None
        if "loglike" in want:
            ll, dh, hh = np.zeros(B), np.zeros(B), np.zeros(B)
            ds, w = _f64(data_spec), _f64(weight)
        rc = self.lib.orc_chain(B, N, M, lp, mp, _p(amp), _p(phase), _p(ang[0]), _p(ang[1]),
                                _p(ang[2]), _p(iota), _p(phi), _p(psi), _p(e0), t0, dt, order,
                                _p(lam), _p(beta_sky), C.byref(o), margin_y, generation, out_kind,
                                margin_lo, margin_hi, n_lo, n_hi, _p(hp), _p(hc), _p(y), _p(tdi),
                                _p(ds), _p(w), kmin, kmax, _p(ll), _p(dh), _p(hh))
        assert rc == 0, rc
        return {"hplus": hp, "hcross": hc, "y": y, "tdi": tdi, "loglike": ll, "dh": dh, "hh": hh}
