#!/usr/bin/env python
"""bench.py -- log-likelihood evaluations per second of the whole hot path (S1..S5) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

Workload (BASELINE.json `metric`): N = 2^20 samples at dt = 5 s, batch 64 precessing walkers
with the five-mode set on KEPLER1 orbits (configs[2]), TDI-2 A,E,T at Lagrange order 31,
forward FFT and the noise-weighted inner product against the zero-noise injection of walker 0
with the configs[3] PSD and band.  One step = one pass of S1..S5 over the batch.  Inputs are
seeded and synthetic (paper_2501_08261_b200/synth.py).

Prints ONE JSON line (see DESIGN.md section 8 for every key).  With N > 1 GPUs (torchrun) every
rank runs its own batch of 64 walkers -- walkers are independent, there is no data-path
collective -- and the value is the aggregate over ranks ("scaling": "weak").
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "loglike evals/sec (2^20 samples, dt=5 s, batch 64)"
UNIT = "evals/s"
WORKLOAD = "configs[2] precessing batch: B=64, N=2^20, dt=5 s, 5 modes, KEPLER1 orbits, TDI-2 AET order 31, + configs[3] PSD/band log L"
CONFIG_ID = 3
ORDER = 31

# Algorithmic fp64 work per walker-sample, in DFMA-equivalent
# instructions (DADD, DMUL, DFMA each count 1; flops = 2 x this).
# 9 evaluation times, each a fused coefficient sweep + two dot products over (p+1)/2 node pairs
# at 11 ops per pair (4 stencil FMAs + 7 for the two coefficients; the first pair saves one),
# plus the per-walker projections, delays and six divisions-free link combinations.  The
# walker-independent orbit evaluation is NOT credited.  The kernel executes 1762 (ncu).
K2_SWEEP = 9 * (11 * (ORDER + 1) // 2 - 1)
K2_GEOM = 150
K2_OPS = K2_SWEEP + K2_GEOM            # 1725 ops = 3450 flop per walker-sample
K2_BYTES = 16 + 48                     # h+,hx in, six links out
# dram__bytes_read.sum + dram__bytes_write.sum of one k2 launch at this workload
# (ncu --set full capture summarised in profiles/r2_s2.md: 1.08 GB read + 3.17 GB written)
K2_TRAFFIC_BYTES = 4.24e9
# K3 (TDI-2, A,E,T): 12 (channel, series) pairs x 44 merged-stencil taps = 528 MACs per walker-sample
# (the 8x8x4 tiles of the banded product issue 624); 48 B of links in, 24 B out
K3_OPS = 528
K3_BYTES = 48 + 24
K1_OPS_EXECUTED = 334                  # fp64 instructions per sample of the five-mode kernel (ncu)


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--batch", type=int, default=64, help=argparse.SUPPRESS)
    ap.add_argument("--log2n", type=int, default=20, help=argparse.SUPPRESS)
    ap.add_argument("--no-e2e", action="store_true", help=argparse.SUPPRESS)
    ap.add_argument("--no-cpu-baseline", action="store_true", help=argparse.SUPPRESS)
    return ap.parse_args()


# ----------------------------------------------------------------------------- helpers
class ClockSampler:
    """nvidia-smi clocks / throttle reasons of one GPU, sampled every 200 ms in the background."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "50"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, smax, power, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            parts = [x.strip() for x in line.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0]))
                smax.append(float(parts[1]))
                power.append(float(parts[2]))
            except ValueError:
                continue
            for nm, v in zip(names, parts[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(smax)),
                       power_w_max=float(max(power)), reasons=sorted(reasons), samples=len(sm))
        return out


def shard_walkers(total_walkers: int, world: int, rank: int):
    """Contiguous block of walkers owned by `rank` (the N>1 path: no data-path collective)."""
    per = total_walkers // world
    rem = total_walkers % world
    lo = rank * per + min(rank, rem)
    return lo, lo + per + (1 if rank < rem else 0)


def dist_max(value: float, dist=None, device=None) -> float:
    """max over ranks of a python float (identity without torch.distributed)."""
    if dist is None or not dist.is_initialized():
        return value
    import torch
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def oracle_sample_rate(inp, data, weight, kmin, kmax, window=None, walkers=1):
    """Time the fp64 CPU oracle, as it stands, on a bounded sample of the workload:
    S1..S3 for `window` output samples of walker 0, then S4+S5 (three full-length FFTs + inner
    product) for one walker.  Returns (evals_per_s, description, threads)."""
    from oracle.binding import Oracle
    orc = Oracle("d")
    N = inp["N"]
    window = N if window is None else min(window, N)
    nwalk = min(walkers, int(inp["amp"].shape[0]))
    n = lambda k: None if inp[k] is None else inp[k][:nwalk].contiguous().cpu().numpy()
    lo = (N - window) // 2
    t0 = time.perf_counter()
    orc.chain(inp["l"], inp["m"], n("amp"), n("phase"), n("iota"), n("phi"), n("psi"), n("lam"), n("beta_sky"),
              inp["orbit"], inp["t0"], inp["dt"], inp["order"], inp["margin_y"], 20, 1, inp["margin_lo"],
              inp["margin_hi"], alpha=n("alpha"), beta=n("beta"), gamma=n("gamma"), n_lo=lo, n_hi=lo + window,
              want=("tdi",))
    t_win = time.perf_counter() - t0
    tdi = np.zeros((nwalk, 3, N))
    tdi[:, :, lo:lo + window] = 1e-22
    t0 = time.perf_counter()
    orc.loglike(tdi, data, weight, kmin, kmax)
    t_fft = time.perf_counter() - t0
    per_eval = (t_win * (N / window) + t_fft) / nwalk
    desc = (f"oracle (fp64 build, OpenMP) on {nwalk} walker(s): S1-S3 on {window} of {N} output samples each "
            f"({t_win:.2f} s, scaled by N/{window}) + S4/S5 at full length ({t_fft:.2f} s)")
    return 1.0 / per_eval, desc, orc.num_threads()


# ----------------------------------------------------------------------------- reference arm
def run_reference(args):
    """--impl reference: the oracle timed on the host cores (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_2501_08261_b200 import synth
    from oracle.binding import Oracle
    N = 1 << args.log2n
    inp = synth.make_inputs(CONFIG_ID, B=1, N=N)
    kmin, kmax = synth.likelihood_band(N, inp["dt"])
    orc = Oracle("d")
    w = orc.psd_weights(N, inp["dt"], synth.NOISE["acc"], synth.NOISE["oms"], synth.NOISE["arm_s"], 20)
    data = np.zeros((3, N // 2 + 1, 2))
    vals, desc, threads = [], "", 1
    for i in range(args.warmup + args.steps):
        v, desc, threads = oracle_sample_rate(inp, data, w, kmin, kmax, window=1 << 17)
        if i >= args.warmup:
            vals.append(v)
    value = float(len(vals) / sum(1.0 / v for v in vals))
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 / value * 64,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": {"workload": WORKLOAD, "l2": "n/a (CPU)"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle",
                         "note": "unoptimised oracle: literal O(p^2) Lagrange products, gcc -O2", "sample": desc, "extrapolated_from_window": True,
                         "measured_s_per_step": float(np.mean([1.0 / v for v in vals]) * (1 << 17) / N)},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


# ----------------------------------------------------------------------------- our arm
def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2501_08261_b200 import lib, synth

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    device = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=device)
    lib.load()

    B, N = args.batch, 1 << args.log2n
    # weak scaling: every rank owns a full batch of B walkers (global batch = world * B);
    # rank r uses seed offset r so the ranks hold different walkers of the same population
    inp = synth.make_inputs(CONFIG_ID, device=device, B=B, N=N, seed=synth.SEED0 + CONFIG_ID + 1000 * rank)
    dt, t0 = inp["dt"], inp["t0"]
    kmin, kmax = synth.likelihood_band(N, dt)
    w_host = lib.psd_weights(N, dt, synth.NOISE["acc"], synth.NOISE["oms"], synth.NOISE["arm_s"], 20)
    weight = torch.from_numpy(w_host).to(device)
    nf = N // 2 + 1
    f64 = torch.float64
    hp = torch.empty((B, N), dtype=f64, device=device)
    hc = torch.empty_like(hp)
    y = torch.empty((B, 6, N), dtype=f64, device=device)
    tdi = torch.empty((B, 3, N), dtype=f64, device=device)
    ll = torch.empty(B, dtype=f64, device=device)
    dh = torch.empty(B, dtype=f64, device=device)
    hh = torch.empty(B, dtype=f64, device=device)
    plan = lib.Plan(B, N)
    g = lambda k: inp[k]

    def s1():
        lib.modes_to_pol(B, N, inp["l"], inp["m"], g("amp"), g("phase"), g("alpha"), g("beta"), g("gamma"),
                         g("iota"), g("phi"), g("psi"), None, hp, hc)

    def s2():
        lib.link_response(B, N, t0, dt, ORDER, inp["margin_y"], hp, hc, g("lam"), g("beta_sky"), inp["orbit"], y)

    def s3():
        lib.tdi2(B, N, t0, dt, ORDER, 20, 1, inp["margin_lo"], inp["margin_hi"], y, inp["orbit"], tdi)

    # zero-noise injection: spectrum of walker 0
    s1(); s2(); s3()
    spec = torch.empty((B, 3, nf, 2), dtype=f64, device=device)
    lib.spectrum(plan, B, N, tdi, spec)
    data = spec[0].contiguous()
    del spec
    torch.cuda.synchronize()

    def s45():
        lib.loglike(plan, B, N, tdi, data, weight, kmin, kmax, ll, dh, hh)

    # fp64 ALU peak, measured in this run (sustained ~1 s, all SMs): the roofline denominator
    sink = torch.empty(148 * 8 * 256, dtype=f64, device=device)
    lib.probe_dfma(20000, 148 * 8, 256, sink)
    iters = 400000
    ms = lib.probe_dfma(iters, 148 * 8, 256, sink)
    dfma_peak_tflops = 2 * 8 * iters * 148 * 8 * 256 / (ms * 1e-3) / 1e12

    # do the DFMA pipe (K1, K2) and the fp64 tensor path (K3) run side by side?  8 + 8 warps per SM
    pipes = {}
    for name, (nf_w, nm_w) in (("dfma_only", (8, 0)), ("dmma_only", (0, 8)), ("both", (8, 8))):
        lib.probe_fp64_pipes(2000, 148, nf_w, nm_w, sink)
        pms = lib.probe_fp64_pipes(100000, 148, nf_w, nm_w, sink)
        pipes[name] = {"ms": pms, "tflops": 2 * 100000 * 148 * (256 * nf_w + 1024 * nm_w) / (pms * 1e-3) / 1e12}
    pipes["reading"] = "times add: one fp64 resource" if pipes["both"]["ms"] > 0.9 * (pipes["dfma_only"]["ms"] + pipes["dmma_only"]["ms"]) else "overlap"

    # issue rate of fp64 instructions by the number of distinct register operands: a DFMA that
    # reads three fresh registers issues every 3 cycles, not 2; "k2_sweep_only" is the node-pair recurrence of
    # K2's sweep on register data, i.e. what that instruction mix can reach with no loads at all
    operands = {}
    for name, (pat, per_round) in (("fma_1_register_operand", (0, 8)), ("mul_2_register_operands", (1, 8)),
                                   ("fma_2_fresh_1_repeated", (2, 8)), ("fma_3_register_operands", (3, 8)),
                                   ("k2_sweep_only", (4, 352))):
        lib.probe_fp64_operands(pat, 2000, 148 * 4, sink)
        it_o = 200000 if pat < 4 else 5000
        oms = lib.probe_fp64_operands(pat, it_o, 148 * 4, sink)
        operands[name] = {"ms": oms, "tflops_equiv": 2 * per_round * it_o * 148 * 4 * 128 / (oms * 1e-3) / 1e12}
    for v in operands.values():
        v["frac_of_dfma_peak"] = v["tflops_equiv"] / dfma_peak_tflops

    stages = [("S1_modes_to_pol", s1), ("S2_link_response", s2), ("S3_tdi2", s3), ("S45_fft_loglike", s45)]
    for _ in range(max(args.warmup, 3)):
        for _, fn in stages:
            fn()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    sampler = ClockSampler(local_rank) if rank == 0 else None
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(len(stages) + 1)] for _ in range(args.steps)]
    torch.cuda.synchronize()
    for k in range(args.steps):
        ev[k][0].record()
        for i, (_, fn) in enumerate(stages):
            fn()
            ev[k][i + 1].record()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    clocks = sampler.stop() if sampler else None
    total_ms = ev[0][0].elapsed_time(ev[-1][-1])
    total_ms = dist_max(total_ms, dist if world > 1 else None, device)
    stage_ms = {nm: float(np.mean([ev[k][i].elapsed_time(ev[k][i + 1]) for k in range(args.steps)]))
                for i, (nm, _) in enumerate(stages)}
    ms_per_step = total_ms / args.steps
    value = world * B / (ms_per_step * 1e-3)
    loglike0 = float(ll[0].item())

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- the same step through the one-call API (lisa_td_loglike_from_modes: S1..S5 from device inputs)
    ws_fm = torch.empty(lib.loglike_from_modes_workspace_bytes(B, N) // 8, dtype=f64, device=device)
    ll_fm = torch.empty(B, dtype=f64, device=device)

    def one_call():
        lib.loglike_from_modes(plan, B, N, inp["l"], inp["m"], g("amp"), g("phase"), g("alpha"), g("beta"), g("gamma"),
                               g("iota"), g("phi"), g("psi"), g("lam"), g("beta_sky"), t0, dt, ORDER, inp["margin_y"], 20,
                               inp["margin_lo"], inp["margin_hi"], inp["orbit"], data, weight, kmin, kmax, ll_fm, None, None,
                               ws_fm)
    for _ in range(3):
        one_call()
    oc = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    oc[0].record()
    for _ in range(5):
        one_call()
    oc[1].record()
    torch.cuda.synchronize()
    one_call_info = {"ms_per_step": oc[0].elapsed_time(oc[1]) / 5, "api": "lisa_td_loglike_from_modes",
                     "bit_identical_to_stagewise": bool(torch.equal(ll_fm, ll))}
    del ws_fm

    # ---- batched finite-difference Fisher matrix, D = 15
    # parameters = 16 walkers (centre + 15 perturbed; the first 16 walkers of the batch, which
    # are 1e-3 perturbations of walker 0, stand in for them) through S1..S3 + lisa_td_fisher
    D = 15
    fis = torch.empty((D, D), dtype=f64, device=device)
    delta = np.full(D, 1e-3)

    def fisher_step():
        lib.modes_to_pol(D + 1, N, inp["l"], inp["m"], g("amp"), g("phase"), g("alpha"), g("beta"), g("gamma"),
                         g("iota"), g("phi"), g("psi"), None, hp, hc)
        lib.link_response(D + 1, N, t0, dt, ORDER, inp["margin_y"], hp, hc, g("lam"), g("beta_sky"), inp["orbit"], y)
        lib.tdi2(D + 1, N, t0, dt, ORDER, 20, 1, inp["margin_lo"], inp["margin_hi"], y, inp["orbit"], tdi)
        lib.fisher(plan, D, N, tdi, delta, weight, kmin, kmax, fis)
    for _ in range(3):
        fisher_step()
    fe = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
    torch.cuda.synchronize()
    fe[0].record()
    for _ in range(5):
        fisher_step()
    fe[1].record()
    for _ in range(5):
        lib.fisher(plan, D, N, tdi, delta, weight, kmin, kmax, fis)
    fe[2].record()
    torch.cuda.synchronize()
    # ---- the paper's 10 s -> 5 s trick: S1 on N/2+1 coarse samples
    # (every other sample of the same inputs) + lisa_td_link_response_up2
    Nc = N // 2 + 1
    cz = lambda k: torch.cat([inp[k][..., ::2], inp[k][..., -1:]], dim=-1).contiguous()
    c_in = {k: cz(k) for k in ("amp", "phase", "alpha", "beta", "gamma")}
    hpc = torch.empty((B, Nc), dtype=f64, device=device)
    hcc = torch.empty_like(hpc)

    def up2_step():
        lib.modes_to_pol(B, Nc, inp["l"], inp["m"], c_in["amp"], c_in["phase"], c_in["alpha"], c_in["beta"],
                         c_in["gamma"], g("iota"), g("phi"), g("psi"), None, hpc, hcc)
        lib.link_response_up2(B, N, t0, dt, ORDER, inp["margin_y"], hpc, hcc, g("lam"), g("beta_sky"), inp["orbit"], y)
    for _ in range(3):
        up2_step()
    ue = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    ue[0].record()
    for _ in range(5):
        up2_step()
    ue[1].record()
    torch.cuda.synchronize()
    up2_info = {"ms_s1_coarse_plus_s2_up2": ue[0].elapsed_time(ue[1]) / 5,
                "ms_s1_plus_s2_full_rate": stage_ms["S1_modes_to_pol"] + stage_ms["S2_link_response"],
                "cite": "PAPER.md:243 (10 s sampling, linear interpolation), DESIGN.md reading A20"}
    del c_in, hpc, hcc
    # ---- SURVEY 8(f) f4, second half: channel subsets A / AE: S4 + S5 on fewer channels
    ch_info = {"ms_s45_AET": stage_ms["S45_fft_loglike"], "cite": "PAPER.md:362"}
    for n_ch, name in ((1, "ms_s45_A"), (2, "ms_s45_AE")):
        for _ in range(3):
            lib.loglike_channels(plan, B, N, n_ch, tdi, data, weight, kmin, kmax, ll, dh, hh)
        ce = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        ce[0].record()
        for _ in range(5):
            lib.loglike_channels(plan, B, N, n_ch, tdi, data, weight, kmin, kmax, ll, dh, hh)
        ce[1].record()
        torch.cuda.synchronize()
        ch_info[name] = ce[0].elapsed_time(ce[1]) / 5
    # ---- first-order light travel times + TDI delays chained along the light path
    # (reading A22): S2 and S3 with that delay model (restores y, tdi of the default model after)
    orb22 = dict(inp["orbit"], tt_order=1, nested=1)

    def nested_s2():
        lib.link_response(B, N, t0, dt, ORDER, inp["margin_y"], hp, hc, g("lam"), g("beta_sky"), orb22, y)

    def nested_s3():
        lib.tdi2(B, N, t0, dt, ORDER, 20, 1, inp["margin_lo"], inp["margin_hi"], y, orb22, tdi)
    for _ in range(3):
        nested_s2(); nested_s3()
    ne = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
    ne[0].record()
    for _ in range(5):
        nested_s2()
    ne[1].record()
    for _ in range(5):
        nested_s3()
    ne[2].record()
    torch.cuda.synchronize()
    nested_info = {"ms_s2_tt_order1": ne[0].elapsed_time(ne[1]) / 5, "ms_s3_chained": ne[1].elapsed_time(ne[2]) / 5,
                   "ms_s2_default": stage_ms["S2_link_response"], "ms_s3_default": stage_ms["S3_tdi2"],
                   "cite": "PAPER.md:163, 380-384; DESIGN.md reading A22"}
    # ---- "with p = 1 (the paper's linear interpolation) also timed"
    def o1_s2():
        lib.link_response(B, N, t0, dt, 1, inp["margin_y"], hp, hc, g("lam"), g("beta_sky"), inp["orbit"], y)

    def o1_s3():
        lib.tdi2(B, N, t0, dt, 1, 20, 1, inp["margin_lo"], inp["margin_hi"], y, inp["orbit"], tdi)
    for _ in range(3):
        o1_s2(); o1_s3()
    oe = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
    oe[0].record()
    for _ in range(5):
        o1_s2()
    oe[1].record()
    for _ in range(5):
        o1_s3()
    oe[2].record()
    torch.cuda.synchronize()
    o1_ms2, o1_ms3 = oe[0].elapsed_time(oe[1]) / 5, oe[1].elapsed_time(oe[2]) / 5
    order1_info = {"ms_s2": o1_ms2, "ms_s3": o1_ms3,
                   "s2_hbm_gbs": 64.0 * B * N / (o1_ms2 * 1e-3) / 1e9, "s3_hbm_gbs": 72.0 * B * N / (o1_ms3 * 1e-3) / 1e9,
                   "hbm_bytes_per_walker_sample": {"s2": 64, "s3": 72},
                   "cite": "PAPER.md:209 (linear interpolation); SURVEY 8(d)"}
    # ---- the fused response+TDI kernel north_star sketches, bounded by measurement:
    # a block that keeps the six links of a time tile in shared memory must compute them on the tile PLUS the
    # reach of the merged TDI stencils (51 samples at order 31, generation 2).  At the largest tile whose links
    # fit in shared memory for 8 walkers (256 outputs -> 307 link samples) its link-response phase is the
    # committed K2 on 307/256 as many samples; its TDI phase is the same banded DMMA product as k3_tdi_mma.
    Nf = ((N * 307 + 255) // 256 + 1) // 2 * 2
    hp_f = torch.zeros((B, Nf), dtype=f64, device=device)
    hc_f = torch.zeros((B, Nf), dtype=f64, device=device)
    hp_f[:, :N] = hp
    hc_f[:, :N] = hc
    y_f = torch.empty((B, 6, Nf), dtype=f64, device=device)

    def fused_k2_phase():
        lib.link_response(B, Nf, t0, dt, ORDER, inp["margin_y"], hp_f, hc_f, g("lam"), g("beta_sky"), inp["orbit"], y_f)
    for _ in range(3):
        fused_k2_phase()
    fb = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    fb[0].record()
    for _ in range(5):
        fused_k2_phase()
    fb[1].record()
    torch.cuda.synchronize()
    ms_k2_fused = fb[0].elapsed_time(fb[1]) / 5
    del hp_f, hc_f, y_f
    fused_info = {"ms_k2_on_tile_plus_stencil_reach": ms_k2_fused, "ms_k2": stage_ms["S2_link_response"],
                  "ms_k3": stage_ms["S3_tdi2"], "ms_unfused_k2_plus_k3": stage_ms["S2_link_response"] + stage_ms["S3_tdi2"],
                  "ms_fused_lower_bound": ms_k2_fused + stage_ms["S3_tdi2"],
                  "reading": "lower bound of a fused kernel with 256-output tiles = K2 on 307/256 of the samples + the same DMMA "
                             "product; the HBM round trip it would save (6.4 GB) is hidden under fp64 work in the unfused path",
                  "cite": "north_star 'fused TDI2 delay-and-sum kept in shared memory'; DESIGN.md section 9"}
    s2(); s3()
    torch.cuda.synchronize()
    fisher_info = {"D": D, "walkers": D + 1, "ms_per_matrix": fe[0].elapsed_time(fe[1]) / 5,
                   "ms_fft_plus_k6": fe[1].elapsed_time(fe[2]) / 5,
                   "cite": "PAPER.md:249 (first-order finite differences), DESIGN.md reading A19"}

    # ---- roofline of the dominant kernel (S2, link response)
    k2_ms = stage_ms["S2_link_response"]
    ws = B * N
    achieved = 2 * K2_OPS * ws / (k2_ms * 1e-3) / 1e12
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except OSError:
        pass
    hbm_peak = peaks.get("hbm_gbs", 6650.0)
    roofline = {
        "kernel": "k2_link_response<16,1>", "bound": "alu", "achieved": achieved, "peak": dfma_peak_tflops,
        "unit": "TFLOP/s", "frac": achieved / dfma_peak_tflops, "traffic": K2_TRAFFIC_BYTES,
        "peak_source": "DFMA probe measured in this run (lisa_td_probe_dfma, all SMs, ~1 s); nominal 148 SM x 64 DFMA/clk x 1.965 GHz = 37.2",
        "ops_per_walker_sample": K2_OPS, "ms_per_launch": k2_ms,
        "hbm_achieved_gbs": K2_BYTES * ws / (k2_ms * 1e-3) / 1e9,
        "hbm_peak_gbs": hbm_peak, "hbm_peak_source": "MEASURED_PEAKS.json" if peaks else "fallback",
        "hbm_frac": K2_BYTES * ws / (k2_ms * 1e-3) / 1e9 / hbm_peak,
    }

    k3_ms = stage_ms["S3_tdi2"]
    roofline["other_kernels"] = {
        "k3_tdi (anchor tables + mma + fix-up)": {
            "bound": "alu (fp64 tensor path, same units)", "ms_per_launch": k3_ms, "ops_per_walker_sample": K3_OPS,
            "achieved": 2 * K3_OPS * ws / (k3_ms * 1e-3) / 1e12, "frac": 2 * K3_OPS * ws / (k3_ms * 1e-3) / 1e12 / dfma_peak_tflops,
            "hbm_achieved_gbs": K3_BYTES * ws / (k3_ms * 1e-3) / 1e9},
        "k1_modes_to_pol": {
            "bound": "alu and hbm, about equally", "ms_per_launch": stage_ms["S1_modes_to_pol"],
            "executed_ops_per_sample": K1_OPS_EXECUTED,
            "frac_alu_executed": 2 * K1_OPS_EXECUTED * ws / (stage_ms["S1_modes_to_pol"] * 1e-3) / 1e12 / dfma_peak_tflops,
            "hbm_achieved_gbs": 120.0 * ws / (stage_ms["S1_modes_to_pol"] * 1e-3) / 1e9,
            "hbm_frac": 120.0 * ws / (stage_ms["S1_modes_to_pol"] * 1e-3) / 1e9 / hbm_peak},
        "whole_step": {
            "credited_ops_per_walker_sample": K1_OPS_EXECUTED + K2_OPS + K3_OPS,
            "frac_of_fp64_peak": 2 * (K1_OPS_EXECUTED + K2_OPS + K3_OPS) * ws / (ms_per_step * 1e-3) / 1e12 / dfma_peak_tflops},
    }
    # the 0.76 of K2 credits 1725 ops, 98 % of what the kernel executes; the count SURVEY 8(d) priced
    # (576 stencil FMAs + 100 geometry, without the nine walker-dependent coefficient sets) gives:
    roofline["frac_survey_priced_ops"] = 2 * (576 + 100) * ws / (k2_ms * 1e-3) / 1e12 / dfma_peak_tflops
    # what K2's instruction mix can reach at all: four of the eleven fp64 instructions of a node pair read three
    # fresh registers and issue every 3 cycles (probe above), so the sweep's own ceiling is ~0.85 of the DFMA peak
    roofline["operand_probe"] = operands
    roofline["frac_of_instruction_mix_ceiling"] = roofline["frac"] / operands["k2_sweep_only"]["frac_of_dfma_peak"]

    # ---- end to end through the host API (pinned host buffers, copies inside the timed region)
    e2e = None
    if not args.no_e2e:
        keys = ["amp", "phase", "alpha", "beta", "gamma", "iota", "phi", "psi", "lam", "beta_sky"]
        host = {k: inp[k].cpu().pin_memory() for k in keys}
        data_h, w_h = data.cpu().pin_memory(), weight.cpu().pin_memory()
        out_h = torch.empty(B, dtype=f64).pin_memory()
        # free the device-resident copies first: the pipeline owns its own chunk buffers
        h2d = sum(host[k].numel() for k in keys) * 8 + (data_h.numel() + w_h.numel()) * 8
        pipe = lib.Pipeline(16, N, len(inp["l"]), True)

        def e2e_step():
            lib.pipeline_host(pipe, B, N, inp["l"], inp["m"], host["amp"], host["phase"], host["alpha"],
                              host["beta"], host["gamma"], host["iota"], host["phi"], host["psi"], host["lam"],
                              host["beta_sky"], t0, dt, ORDER, inp["margin_y"], 20, inp["margin_lo"],
                              inp["margin_hi"], inp["orbit"], data_h, w_h, kmin, kmax, out_h)
        e2e_step()
        torch.cuda.synchronize()
        n_e2e = 3
        t_start = time.perf_counter()
        for _ in range(n_e2e):
            e2e_step()
        t_e2e = (time.perf_counter() - t_start) / n_e2e
        assert abs(float(out_h[0]) - loglike0) <= 1e-9 * abs(loglike0), (float(out_h[0]), loglike0)
        e2e = {"value": B / t_e2e, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(B * 8),
               "ms_per_step": t_e2e * 1e3, "api": "lisa_td_pipeline_host (chunks of 16 walkers, copy/compute streams)",
               "steps": n_e2e}
        # the same call with the paper's 10 s sampling of the modes: half the bytes cross PCIe
        cz = lambda t: torch.cat([t[..., ::2], t[..., -1:]], dim=-1).contiguous().pin_memory()
        host_c = {k: cz(host[k]) for k in ("amp", "phase", "alpha", "beta", "gamma")}
        out_c = torch.empty(B, dtype=f64).pin_memory()

        def e2e_up2_step():
            lib.pipeline_host_up2(pipe, B, N, inp["l"], inp["m"], host_c["amp"], host_c["phase"], host_c["alpha"],
                                  host_c["beta"], host_c["gamma"], host["iota"], host["phi"], host["psi"], host["lam"],
                                  host["beta_sky"], t0, dt, ORDER, inp["margin_y"], 20, inp["margin_lo"],
                                  inp["margin_hi"], inp["orbit"], data_h, w_h, kmin, kmax, out_c)
        e2e_up2_step()
        t_start = time.perf_counter()
        for _ in range(n_e2e):
            e2e_up2_step()
        t_up2 = (time.perf_counter() - t_start) / n_e2e
        e2e["up2"] = {"value": B / t_up2, "unit": UNIT, "ms_per_step": t_up2 * 1e3,
                      "h2d_bytes_per_step": int(sum(host_c[k].numel() for k in host_c) * 8 + (data_h.numel() + w_h.numel()) * 8),
                      "api": "lisa_td_pipeline_host_up2 (modes on the 10 s grid, PAPER.md:243; a different, coarser input: not the headline)",
                      "loglike_walker0_rel_diff": abs(float(out_c[0]) - loglike0) / abs(loglike0)}
        del host_c
        pipe.close()

    # ---- the oracle beside it (bounded sample, host cores)
    cpu_baseline = None
    if not args.no_cpu_baseline:
        inp1 = {k: (v[:2].cpu() if isinstance(v, torch.Tensor) else v) for k, v in inp.items()}
        v, desc, threads = oracle_sample_rate(inp1, data.cpu().numpy(), w_host, kmin, kmax, walkers=2)
        cpu_baseline = {"value": v, "unit": UNIT, "cores": threads,
                        "kind": "oracle", "note": "unoptimised oracle: literal O(p^2) Lagrange products, gcc -O2", "sample": desc}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOAD, "global_batch": world * B, "N": N, "dt": dt, "order": ORDER,
                   "l2": "inputs (6.8 GB per step) and every intermediate exceed the 126 MB L2",
                   "parallelism": f"walker-split x{world}, no collective"},
        "samples_per_s": value * N, "stage_ms": stage_ms, "roofline": roofline, "cpu_baseline": cpu_baseline,
        "e2e": e2e, "gpu_launches": 7 * args.steps, "launches_per_step": {
            "k1_modes_to_pol_std5_tma": 1, "k2_link_response": 1, "k3_anchor_tables": 1, "k3_tdi_mma": 1,
            "k3_tdi_fixup": 1, "k5_inner_partial": 1, "k5_inner_final": 1,
            "cufft (library)": "Z2Z length N/2, batch 192 (packed real input)"},
        "clocks": clocks, "loglike_walker0": loglike0, "dfma_peak_tflops_measured": dfma_peak_tflops, "fp64_pipes": pipes,
        "next": {"fisher": fisher_info, "up2": up2_info, "nested": nested_info, "channels": ch_info,
                 "order1": order1_info, "fused_bound": fused_info, "one_call": one_call_info},
    }
    print(json.dumps(line))
    plan.close()
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
