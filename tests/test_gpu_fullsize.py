"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times
(whole batch per call), checked on sampled output windows the oracle computes one by one.

configs[2] (B = 64, N = 2^20, precessing), its log-likelihood (configs[3] PSD / band) and
configs[4] (stress: B = 32, N = 2^22, plus the common laser-noise stream at scale).  The
inputs are generated on the device (same seeded generator) and the sampled walkers' arrays are
copied to the host for the oracle, so both sides see the same bits.  Odd-N cases cover the
scalar load/store and cp.async paths of the kernels.
"""
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


def _gpu_chain_full(lib, inp, B, N):
    f64 = torch.float64
    hp = torch.empty((B, N), dtype=f64, device="cuda")
    hc = torch.empty_like(hp)
    y = torch.empty((B, 6, N), dtype=f64, device="cuda")
    tdi = torch.empty((B, 3, N), dtype=f64, device="cuda")
    lib.modes_to_pol(B, N, inp["l"], inp["m"], inp["amp"], inp["phase"], inp["alpha"], inp["beta"], inp["gamma"],
                     inp["iota"], inp["phi"], inp["psi"], None, hp, hc)
    lib.link_response(B, N, inp["t0"], inp["dt"], inp["order"], inp["margin_y"], hp, hc, inp["lam"],
                      inp["beta_sky"], inp["orbit"], y)
    lib.tdi2(B, N, inp["t0"], inp["dt"], inp["order"], 20, 1, inp["margin_lo"], inp["margin_hi"], y,
             inp["orbit"], tdi)
    torch.cuda.synchronize()
    return hp, hc, y, tdi


def _walker_to_host(inp, b):
    """single-walker copy of the inputs as numpy arrays (same bits)"""
    out = {}
    for k in ("amp", "phase", "alpha", "beta", "gamma", "iota", "phi", "psi", "lam", "beta_sky"):
        out[k] = None if inp[k] is None else inp[k][b:b + 1].contiguous().cpu().numpy()
    return out


def _orc_window(orc, inp, h, lo, hi, **kw):
    return orc.chain(inp["l"], inp["m"], h["amp"], h["phase"], h["iota"], h["phi"], h["psi"], h["lam"],
                     h["beta_sky"], inp["orbit"], inp["t0"], inp["dt"], inp["order"], inp["margin_y"], 20, 1,
                     inp["margin_lo"], inp["margin_hi"], alpha=h["alpha"], beta=h["beta"], gamma=h["gamma"],
                     n_lo=lo, n_hi=hi, **kw)


def _check_windows(orc, orc_d, inp, tdi, B, N, walkers, width, rec=None, config=None):
    """Windows of the output against the long-double oracle.  A window at the start of a months-
    long chirp holds a sub-mHz signal whose TDI output is a ~1e-6 remnant of the links, so its
    error relative to the WINDOW's norm sits at the fp64 rounding floor of any fp64 chain
    (SURVEY P4), not at 1e-11 of the channel.  The bar per window is therefore
    max(1e-11, 4 x floor), floor = the error of the oracle's own fp64 build on the same window
    (same formula, plain loops); the whole-channel 1e-11 bar is asserted by the full-length
    comparison below."""
    windows = [(0, width), (N // 2 - width // 2, N // 2 + width // 2), (N // 3 + 17, N // 3 + 17 + width),
               (N - width, N)]
    for b in walkers:
        h = _walker_to_host(inp, b)
        for lo, hi in windows:
            ref = _orc_window(orc, inp, h, lo, hi, want=("tdi",))["tdi"][0][:, lo:hi]
            ref_d = _orc_window(orc_d, inp, h, lo, hi, want=("tdi",))["tdi"][0][:, lo:hi]
            got = tdi[b, :, lo:hi].cpu().numpy()
            # exact zeros outside the valid region (reading A7)
            if lo < inp["margin_lo"]:
                assert np.all(got[:, :min(hi, inp["margin_lo"]) - lo] == 0.0)
            if hi > N - inp["margin_hi"]:
                assert np.all(got[:, max(N - inp["margin_hi"], lo) - lo:] == 0.0)
            common = max(np.linalg.norm(ref[c]) for c in range(3))
            assert common > 0.0
            for c in range(3):
                err = np.linalg.norm(got[c] - ref[c]) / common
                floor = np.linalg.norm(ref_d[c] - ref[c]) / common
                print(f"walker {b} window [{lo},{hi}) channel {c}: err {err:.2e}, fp64 floor {floor:.2e}")
                if rec is not None:
                    nrm = np.linalg.norm(ref[c])
                    rec(config, f"walker {b} window [{lo},{hi}) order {inp['order']}", "AET"[c],
                        raw=None if nrm == 0 else np.linalg.norm(got[c] - ref[c]) / nrm, common=err, floor=floor,
                        tol=max(TOL_TDI, 4.0 * floor), passed=err < max(TOL_TDI, 4.0 * floor),
                        note="window metric: error and floor relative to the window's common scale; bar = max(1e-11, 4 x floor)")
                assert err < max(TOL_TDI, 4.0 * floor), (b, lo, hi, c, err, floor)


def _check_whole_series(orc, orc_d, inp, tdi, b, N, rec, config, case):
    """one walker over ALL N samples against the long-double oracle: raw rel-L2 per channel (the
    north_star bar), the error relative to the common scale of A, E, T, and the fp64 floor (the
    oracle's own fp64 build).  A and E are asserted raw; T, a 1e-3..1e-5 remnant of X on nearly equal
    arms, against the common scale, with its raw value recorded next to its floor."""
    h = _walker_to_host(inp, b)
    ref = _orc_window(orc, inp, h, 0, N, want=("tdi",))["tdi"][0]
    ref_d = _orc_window(orc_d, inp, h, 0, N, want=("tdi",))["tdi"][0]
    got = tdi[b].cpu().numpy()
    common = max(np.linalg.norm(ref[c]) for c in range(3))
    raw = [float(np.linalg.norm(got[c] - ref[c]) / np.linalg.norm(ref[c])) for c in range(3)]
    com = [float(np.linalg.norm(got[c] - ref[c]) / common) for c in range(3)]
    flo = [float(np.linalg.norm(ref_d[c] - ref[c]) / np.linalg.norm(ref[c])) for c in range(3)]
    print(f"{config} {case}: raw rel-L2 {raw}, vs common scale {com}, fp64 floor {flo}")
    for c in range(3):
        rec(config, case, "AET"[c], raw=raw[c], common=com[c], floor=flo[c], tol=TOL_TDI, passed=raw[c] < TOL_TDI,
            note=None if raw[c] < TOL_TDI else "raw above the bar, at the fp64 floor of this channel: asserted against the common scale")
    assert raw[0] < TOL_TDI and raw[1] < TOL_TDI
    assert com[2] < TOL_TDI
    assert raw[2] < max(TOL_TDI, 4.0 * flo[2])   # raw T no worse than four times what ANY fp64 chain loses


def test_config3_full_size_sampled(lib, orc, orc_d, parity_record):
    """configs[2]: B = 64, N = 2^20, the bench.py workload and launch configuration.  Walkers 0
    and 63 are compared over ALL N samples (rel-L2 per channel, the north_star bar), walker 21
    on sampled windows."""
    B, N = 64, 1 << 20
    inp = synth.make_inputs(3, device="cuda", B=B, N=N)
    _, _, _, tdi = _gpu_chain_full(lib, inp, B, N)
    for b in (0, 63):
        _check_whole_series(orc, orc_d, inp, tdi, b, N, parity_record, "configs[2]", f"B=64 N=2^20 walker {b} whole series")
    _check_windows(orc, orc_d, inp, tdi, B, N, walkers=(21,), width=2048, rec=parity_record, config="configs[2]")


def test_order1_full_size_sampled(lib, orc, orc_d, parity_record):
    """the paper's linear interpolation (order 1) at B = 64, N = 2^20: the
    k2_link_response_lin / k3_tdi_mma<1,*> launch configuration the bench times under next.order1"""
    B, N = 64, 1 << 20
    inp = synth.make_inputs(3, device="cuda", B=B, N=N)
    inp["order"] = 1
    _, _, _, tdi = _gpu_chain_full(lib, inp, B, N)
    _check_whole_series(orc, orc_d, inp, tdi, 0, N, parity_record, "configs[2] at order 1", "B=64 N=2^20 walker 0 whole series")
    _check_windows(orc, orc_d, inp, tdi, B, N, walkers=(40, 63), width=2048, rec=parity_record, config="configs[2] at order 1")


def test_config4_full_size_loglike(lib, orc, orc_d, parity_record):
    """configs[3] likelihood at N = 2^20 for two walkers of a full batch-64 launch.  The oracle
    builds its OWN zero-noise injection (walker 0) and its own weights.  Walker 0 -- injection and
    template -- goes through the LONG-DOUBLE build (one full-length chain, about a minute of host
    time); walker 40 is then checked against the fp64 build with the long-double injection."""
    B, N = 64, 1 << 20
    inp = synth.make_inputs(4, device="cuda", B=B, N=N)
    dt = inp["dt"]
    kmin, kmax = synth.likelihood_band(N, dt)
    _, _, _, tdi = _gpu_chain_full(lib, inp, B, N)
    plan = lib.Plan(B, N)
    spec = torch.empty((B, 3, N // 2 + 1, 2), dtype=torch.float64, device="cuda")
    lib.spectrum(plan, B, N, tdi, spec)
    data_gpu = spec[0].contiguous()
    del spec
    w_gpu = torch.from_numpy(lib.psd_weights(N, dt, synth.NOISE["acc"], synth.NOISE["oms"], synth.NOISE["arm_s"], 20)).cuda()
    ll, dh, hh = (torch.empty(B, dtype=torch.float64, device="cuda") for _ in range(3))
    lib.loglike(plan, B, N, tdi, data_gpu, w_gpu, kmin, kmax, ll, dh, hh)
    torch.cuda.synchronize()
    w = orc.psd_weights(N, dt, synth.NOISE["acc"], synth.NOISE["oms"], synth.NOISE["arm_s"], 20)
    h0 = _walker_to_host(inp, 0)
    tdi0 = _orc_window(orc, inp, h0, 0, N, want=("tdi",))["tdi"]          # long double, rounded once at the end
    data = orc.spectrum3(tdi0[0])
    ref0 = dict(zip(("loglike", "dh", "hh"), orc.loglike(tdi0, data, w, kmin, kmax)))
    hb = _walker_to_host(inp, 40)
    ref40 = _orc_window(orc_d, inp, hb, 0, N, want=("loglike",), data_spec=data, weight=w, kmin=kmin, kmax=kmax)
    for b, ref, truth in ((0, ref0, "long double"), (40, ref40, "fp64 build")):
        for got, key in ((ll, "loglike"), (dh, "dh"), (hh, "hh")):
            err = abs(got[b].item() - ref[key][0]) / abs(ref[key][0])
            print(b, key, err)
            parity_record("configs[3]", f"B=64 N=2^20 walker {b} ({truth} oracle)", key, raw=err, tol=TOL_LL, passed=err < TOL_LL)
            assert err < TOL_LL, (b, key, err)
    plan.close()


def test_config2_full_size_single_source(lib, orc, orc_d, parity_record):
    """configs[1]: one source, N = 2^20, aligned spin (no Euler angles), KEPLER1, TDI-2 A,E,T:
    the whole series against the long-double oracle (the batch-1 launch configuration)."""
    B, N = 1, 1 << 20
    inp = synth.make_inputs(2, device="cuda", B=B, N=N)
    assert inp["alpha"] is None
    _, _, _, tdi = _gpu_chain_full(lib, inp, B, N)
    _check_whole_series(orc, orc_d, inp, tdi, 0, N, parity_record, "configs[1]", "B=1 N=2^20 whole series")


def test_config4_batch_256(lib, orc_d, parity_record):
    """configs[3] as stated: batch 256 in ONE launch per stage (48 GiB of arrays on the device);
    log L of the first, a middle and the last walker against the oracle's own chain."""
    B, N = 256, 1 << 20
    inp = synth.make_inputs(4, device="cuda", B=B, N=N)
    dt = inp["dt"]
    kmin, kmax = synth.likelihood_band(N, dt)
    hp, hc, y, tdi = _gpu_chain_full(lib, inp, B, N)
    del hp, hc, y
    plan = lib.Plan(B, N)
    spec = torch.empty((1, 3, N // 2 + 1, 2), dtype=torch.float64, device="cuda")
    lib.spectrum(plan, 1, N, tdi[:1], spec)
    data_gpu = spec[0].contiguous()
    w_gpu = torch.from_numpy(lib.psd_weights(N, dt, synth.NOISE["acc"], synth.NOISE["oms"], synth.NOISE["arm_s"], 20)).cuda()
    ll, dh, hh = (torch.empty(B, dtype=torch.float64, device="cuda") for _ in range(3))
    lib.loglike(plan, B, N, tdi, data_gpu, w_gpu, kmin, kmax, ll, dh, hh)
    torch.cuda.synchronize()
    assert torch.isfinite(ll).all()
    w = orc_d.psd_weights(N, dt, synth.NOISE["acc"], synth.NOISE["oms"], synth.NOISE["arm_s"], 20)
    h0 = _walker_to_host(inp, 0)
    data = orc_d.spectrum3(_orc_window(orc_d, inp, h0, 0, N, want=("tdi",))["tdi"][0])
    for b in (0, 131, 255):
        hb = _walker_to_host(inp, b)
        ref = _orc_window(orc_d, inp, hb, 0, N, want=("loglike",), data_spec=data, weight=w, kmin=kmin, kmax=kmax)
        for got, key in ((ll, "loglike"), (dh, "dh"), (hh, "hh")):
            err = abs(got[b].item() - ref[key][0]) / abs(ref[key][0])
            print(b, key, err)
            parity_record("configs[3]", f"B=256 N=2^20 walker {b} (fp64 build oracle)", key, raw=err, tol=TOL_LL, passed=err < TOL_LL)
            assert err < TOL_LL, (b, key, err)
    plan.close()
    del tdi, inp
    torch.cuda.empty_cache()


def test_config5_stress_sampled(lib, orc, orc_d, parity_record):
    """configs[4]: N = 2^22, B = 32, precessing, Kepler arms; plus the common laser-noise stream
    through the link helper and TDI-2 at full length (reading A12, P6: absolute tolerance)."""
    B, N = 32, 1 << 22
    inp = synth.make_inputs(5, device="cuda", B=B, N=N)
    _, _, _, tdi = _gpu_chain_full(lib, inp, B, N)
    _check_windows(orc, orc_d, inp, tdi, B, N, walkers=(0, 31), width=1024, rec=parity_record, config="configs[4]")
    del tdi
    # laser pass
    p = synth.laser_stream(N)
    margin = 32
    y = torch.empty((6, N), dtype=torch.float64, device="cuda")
    lib.laser_links(N, 0.0, inp["dt"], 31, margin, torch.from_numpy(p).cuda(), inp["orbit"], y)
    out = torch.empty((1, 3, N), dtype=torch.float64, device="cuda")
    mlo, mhi = margin + 32, margin + 16
    lib.tdi2(1, N, 0.0, inp["dt"], 31, 20, 0, mlo, mhi, y.view(1, 6, N), inp["orbit"], out)
    torch.cuda.synchronize()
    yref = orc.laser_links(p, inp["orbit"], 0.0, inp["dt"], 31, margin)
    rms = np.sqrt(np.mean(yref ** 2))
    e_links = np.max(np.abs(y.cpu().numpy() - yref)) / rms
    parity_record("configs[4]", "laser stream N=2^22, six links, max abs error / rms(y_laser) (P6: absolute bar)", "y_laser",
                  raw=e_links, tol=1e-11, passed=e_links < 1e-11)
    assert e_links < 1e-11
    for lo in (0, N // 2, N - 4096):
        ref = orc.tdi(yref[None], inp["orbit"], 0.0, inp["dt"], 31, 20, 0, mlo, mhi, n_lo=lo, n_hi=lo + 4096)
        got = out[0, :, lo:lo + 4096].cpu().numpy()
        e_tdi = np.max(np.abs(got - ref[0][:, lo:lo + 4096])) / rms
        parity_record("configs[4]", f"laser stream through TDI-2, window [{lo},{lo + 4096}), max abs error / rms(y_laser)", "XYZ",
                      raw=e_tdi, tol=1e-11, passed=e_tdi < 1e-11)
        assert e_tdi < 1e-11
    # TDI-2 suppresses the common laser noise below 20 mHz (windowed amplitude ratio)
    seg = slice(N // 2, N // 2 + (1 << 16))
    win = np.kaiser(1 << 16, 30.0)
    f = np.fft.rfftfreq(1 << 16, inp["dt"])
    band = (f > 1e-3) & (f < 2e-2)
    X = np.abs(np.fft.rfft(win * out[0, 0, seg].cpu().numpy()))[band]
    Y = np.abs(np.fft.rfft(win * yref[0, seg]))[band]
    assert np.sqrt(np.mean(X ** 2) / np.mean(Y ** 2)) < 1e-5


@pytest.mark.parametrize("N", [4097, 5001])
def test_odd_length_chain(lib, orc, N):
    """Odd N: scalar loads/stores in K1/K2 and the zero-filling cp.async path of K3."""
    B = 3
    inp = synth.make_inputs(3, device="cuda", B=B, N=N)
    hp, hc, y, tdi = _gpu_chain_full(lib, inp, B, N)
    for b in range(B):
        h = _walker_to_host(inp, b)
        ref = _orc_window(orc, inp, h, 0, N, want=("h", "y", "tdi"))
        assert np.linalg.norm(hp[b].cpu().numpy() - ref["hplus"][0]) / np.linalg.norm(ref["hplus"][0]) < 3e-15
        for l in range(6):
            assert np.linalg.norm(y[b, l].cpu().numpy() - ref["y"][0, l]) / np.linalg.norm(ref["y"][0, l]) < 2e-13
        common = max(np.linalg.norm(ref["tdi"][0, c]) for c in range(3))
        for c in range(3):
            assert np.linalg.norm(tdi[b, c].cpu().numpy() - ref["tdi"][0, c]) / common < TOL_TDI
