#!/usr/bin/env python
"""bench.py -- headline measurement: spin-s SHT / Wigner transforms on one B200 (and N independent ranks).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--no-sweep] [--shard rings]

A "step" is one pass of the whole hot path over one synthetic input: an inverse transform (flm -> map) followed by a
forward transform (map -> flm).  The headline workload is BASELINE.json configs[4], first half: spin-0 complex SHT, MW
sampling, L = 8192, fp64 -- the largest single-GPU configuration, and the one the north_star target ("fused kernel >= 40 % of
FP64 peak at L >= 2048") is stated on.  `value` is transform pairs per second over all ranks with inputs resident in HBM;
`e2e` is the same through the host-buffer C-ABI calls (H2D / D2H inside the timed region).  `roofline` is the fused
recursion + contraction kernel of the forward transform against the FP64 FMA-pipe peak measured in the same process;
`sweep` carries the metric of BASELINE.json itself -- ms (hot / fft / staging), fraction of FP64 peak, and GB/s of the FFT and
staging stages -- versus L for MW, for HEALPix, SO(3), the fp32 variant and the batched (DMMA) configuration.
`cpu_baseline` is the CPU oracle on a bounded sample.  One JSON line on stdout (rank 0).
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

WORKLOAD = dict(L=8192, spin=0, seed=4)
UNIT = "transform_pairs/s"
# dram__bytes_read.sum + dram__bytes_write.sum of the forward theta kernel, per launch, from the ncu --set full captures under
# profiles/ (file named beside each); key (L, spin, batch).  Not measurable inside this process: null for other workloads.
NCU_TRAFFIC_BYTES = {
    (1024, 2, 1): (127.888128e6 + 10.841600e6, "profiles/r2b_theta_kernels.md"),
    (2048, 0, 1): (1.801608e9 + 336.916480e6, "profiles/r2d_theta_kernels.md"),
    (4096, 0, 1): (31.937931e9 + 3.441399e9, "profiles/r2d_theta_kernels.md"),
    (8192, 0, 1): (260.120313e9 + 31.275355e9, "profiles/r2d_theta_kernels.md"),
    (2048, 0, 16): (46.052300e9 + 11.329958e9, "profiles/r2_theta_kernels.md"),
}


def metric_name(L, spin):
    return f"SHT fwd+inv transform pairs per second (MW L={L} spin-{spin} fp64, 1 B200)"


def workload_name(L, spin, B=1):
    tag = {(8192, 0, 1): "BASELINE.json configs[4] (first half)", (1024, 2, 1): "BASELINE.json configs[1]",
           (2048, 0, 16): "BASELINE.json configs[4] (second half)"}.get((L, spin, B), "override")
    sig = "1/(l(l+1)) (l >= 2)" if spin == 2 else "1/(l+1)^2"
    return (f"{tag}: spin-{spin} complex SHT, MW sampling L={L} ({L}x{2 * L - 1}), fp64, "
            + (f"batch of {B} maps transformed together, " if B > 1 else "")
            + f"flm complex Gaussian with variance {sig}, inverse + forward per step; the L >= 2048 rows of `sweep` are the "
              "north_star target evidence")


def sigma_for(spin):
    from paper_2311_14670_b200 import synth
    return synth.SIGMA_CMB if spin == 2 else synth.SIGMA_RED


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return json.load(open(p)), "measured"
    return dict(hbm_gbs=6650.0, bf16_tflops=1590.0), "fallback"


class ClockSampler:
    """nvidia-smi clocks/throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu):
        self.gpu, self.proc, self.lines = gpu, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.gpu), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "25"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if self.proc is None:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, smax, pw, reasons = [], [], [], set()
        for ln in self.lines:
            c = [x.strip() for x in ln.split(",")]
            if len(c) < 9:
                continue
            try:
                sm.append(float(c[1])); smax.append(float(c[2])); pw.append(float(c[3]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), c[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return dict(sm_mhz=statistics.median(sm) if sm else None, sm_max_mhz=max(smax) if smax else None,
                    reasons=sorted(reasons), samples=len(sm), power_w_max=max(pw) if pw else None)


_QUAD_TABLE_S = {}     # L -> seconds the oracle takes to build the ring table of its 2L quadrature rings (measured once per process)


def oracle_sample(L, spin, flm, n_cols):
    """Time the CPU oracle (as it stands) on a bounded sample of the workload and extrapolate to one inverse + one forward.

    Sample: the theta steps (Eq. 33 and Eq. 30, the O(L^3) part) of n_cols harmonic orders m spread over [-(L-1), L-1].
    The cost of a column is proportional to L - |m| (the l-recurrence of the oracle's d-functions starts at l = |m|), so the
    sample is scaled by sum_m (L - |m|) / sum_sample (L - |m|).  The inverse runs on all L MW rings.  The oracle's forward runs on
    its 2L quadrature rings, whose ring table (an O(L^2) long-double sum for the weights: 30-120 s at L = 8192) it rebuilds in every
    call: that table is timed ONCE per process (it is needed once per transform, not once per sampled column -- scaling it with the
    columns, as this function did before, overstated the oracle's forward time about five-fold), and the columns are timed on the L
    MW rings (a per-ring cost, so x 2 for the 2L quadrature rings).  forward = table + 2 x scaled columns.  The oracle's ring DFTs are
    deliberately naive O(n^2) sums and are NOT part of the sample (they would take 13 s per ring at L = 8192); the extrapolated time
    therefore flatters the oracle."""
    import oracle as O
    ms = np.unique(np.linspace(-(L - 1), L - 1, n_cols).astype(int))
    scale = float(L * L) / float(np.sum(L - np.abs(ms)))          # sum_{|m| < L} (L - |m|) = L^2
    t0 = time.perf_counter()
    F = O.s2_theta_inverse_columns(L, spin, O.MW, flm, ms)
    t_inv = (time.perf_counter() - t0) * scale
    if L not in _QUAD_TABLE_S:
        t0 = time.perf_counter()
        O.ring_table(O.MW_QUAD, L)
        _QUAD_TABLE_S[L] = time.perf_counter() - t0
    # forward theta step: the values do not matter for timing
    t0 = time.perf_counter()
    O.s2_theta_forward_columns(L, spin, O.MW, np.ascontiguousarray(F), ms)
    t_fwd = _QUAD_TABLE_S[L] + 2.0 * (time.perf_counter() - t0) * scale
    return t_inv, t_fwd, O.threads(), (f"theta steps of {len(ms)} of {2 * L - 1} orders m, scaled by sum(L-|m|): Eq. 33 on the {L} MW rings; Eq. 30 on "
                                       f"the {L} MW rings x 2 (the oracle's forward uses {2 * L} quadrature rings) + its quadrature ring table "
                                       f"({_QUAD_TABLE_S[L]:.1f} s, timed once); naive O(n^2) ring DFTs of the oracle excluded")


REF_COLS = 16          # orders m per step of `--impl reference`: one per thread on the 16-thread GPU box, about 5 s per step at L = 8192, so that
                       # the driver's --steps 20 --warmup 5 run ends in about 3 minutes (plus the quadrature table, once)


def run_reference(args):
    """--impl reference: the CPU oracle on the same config/metric (bounded sample per step)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_2311_14670_b200 import synth
    L, spin = WORKLOAD["L"], WORKLOAD["spin"]
    flm = synth.random_flm(L, spin, seed=WORKLOAD["seed"], sigma=sigma_for(spin))
    times = []
    sample = ""
    for i in range(args.warmup + args.steps):
        t_inv, t_fwd, cores, sample = oracle_sample(L, spin, flm, n_cols=REF_COLS)
        if i >= args.warmup:
            times.append(t_inv + t_fwd)
    t = float(np.mean(times))
    v = 1.0 / t
    print(json.dumps({
        "impl": "reference", "metric": metric_name(L, spin), "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": t * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f80 (long double)", "data": "synthetic",
        "config": {"workload": workload_name(L, spin), "l2": "n/a (CPU)", "parallelism": f"independent x{args.gpus}"},
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def time_stages(plan, x, flush, reps=5):
    """Median per-stage device times (CUDA events recorded inside the library on the launching stream) and the algorithmic
    bytes of the FFT / staging sections of one inverse and one forward transform."""
    plan.enable_timing(True)
    f = plan.inverse(x)
    b = plan.forward(f)
    ti, tf = [], []
    for _ in range(reps):
        flush.zero_(); plan.inverse(x, out=f); ti.append(plan.timings()); bi = plan.stage_bytes()
        flush.zero_(); plan.forward(f, out=b); tf.append(plan.timings()); bf = plan.stage_bytes()
    plan.enable_timing(False)
    med = lambda ts: {k: statistics.median(t[k] for t in ts) for k in ("hot", "fft", "staging", "total")}
    err = float((b - x).abs().max() / x.abs().max())
    return med(ti), med(tf), bi, bf, err


def time_pairs(plan, x, torch, target_ms=40.0):
    """ms per inverse + forward pair through the normal call path (stage timing off, so plans with L <= 512 replay their captured CUDA
    graphs), back to back on the same buffers, CUDA events around the whole loop."""
    f = plan.inverse(x)
    b = plan.forward(f)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

    def loop(n):
        e0.record()
        for _ in range(n):
            plan.inverse(x, out=f); plan.forward(f, out=b)
        e1.record(); e1.synchronize()
        return e0.elapsed_time(e1) / n
    t = loop(3)
    return loop(max(3, min(400, int(target_ms / max(t, 1e-3)))))


def compact(ms, nbytes, flops, peak_tf):
    """One direction of a sweep row: ms per stage, fraction of the arithmetic peak in the hot kernels, GB/s of the HBM-bound stages."""
    gbs = lambda b, t: round(b / (t * 1e-3) / 1e9, 1) if t > 0 else None
    return {"hot_ms": round(ms["hot"], 4), "fft_ms": round(ms["fft"], 4), "staging_ms": round(ms["staging"], 4),
            "frac": round(flops / (ms["hot"] * 1e-3) / 1e12 / peak_tf, 4) if ms["hot"] > 0 else None,
            "fft_gbs": gbs(nbytes["fft"], ms["fft"]), "staging_gbs": gbs(nbytes["staging"], ms["staging"])}


def sweep(api, synth, torch, dev, flush, pk):
    """BASELINE.json's metric: ms (hot / fft / staging) and fraction of FP64 peak vs L for MW, HEALPix, SO(3), plus the fp32 and the
    batched (DMMA) configurations; GB/s of the HBM-bound stages.  `frac` = algorithmic flop / hot time / measured peak."""
    rows = []

    def add(name, plan, x, peak_tf, extra=None):
        mi, mf, bi, bf, err = time_stages(plan, x, flush, reps=3)
        r = {"config": name, "inverse": compact(mi, bi, plan.flops(False), peak_tf), "forward": compact(mf, bf, plan.flops(True), peak_tf),
             "pair_ms": round(time_pairs(plan, x, torch), 4), "roundtrip_err": float(f"{err:.3e}")}
        if extra:
            r.update(extra)
        rows.append(r)

    def mw(L, spin, sigma, seed, **kw):
        return torch.from_numpy(synth.random_flm(L, spin, seed=seed, sigma=sigma)).to(dev)

    for L, spin, sigma, seed, tag in ((64, 0, synth.SIGMA_UNIT, 0, "configs[0] "), (1024, 2, synth.SIGMA_CMB, 1, "configs[1] "),
                                      (2048, 0, synth.SIGMA_RED, 4, ""), (2048, 2, synth.SIGMA_CMB, 1, ""), (4096, 0, synth.SIGMA_RED, 4, "")):
        x = mw(L, spin, sigma, seed)
        P = api.Plan(L, spin, device=dev)
        add(f"{tag}MW spin-{spin} L={L} fp64", P, x, pk["dfma"])
        del P, x
        torch.cuda.empty_cache()
    # configs[4], fp32 variant: complex64 arrays, fp32 recursion + contraction; frac against the measured FFMA peak
    for L in (2048, 8192):
        x = torch.from_numpy(synth.random_flm(L, 0, seed=4, sigma=synth.SIGMA_RED).astype("complex64")).to(dev)
        P = api.Plan(L, 0, device=dev, dtype="f32")
        add(f"configs[4] MW spin-0 L={L} fp32", P, x, pk["ffma"], {"peak": "ffma"})
        del P, x
        torch.cuda.empty_cache()
    # configs[4], second half: 16 maps at L = 2048 transformed together (shared recursion, FP64 DMMA contraction)
    L, B = 2048, 16
    x = torch.from_numpy(np.stack([synth.random_flm(L, 0, seed=4 + i, sigma=synth.SIGMA_RED) for i in range(B)])).to(dev)
    P = api.Plan(L, 0, device=dev, batch=B)
    add(f"configs[4] MW spin-0 L={L} batch {B} (theta_mma_kernel, FP64 DMMA)", P, x, pk["dfma"], {"maps": B})
    del P, x
    torch.cuda.empty_cache()
    # configs[2]: real spin-0 SHT on HEALPix nside = 1024, L = 2048 (forward of the synthesised map: inexact by design)
    nside, L = 1024, 2048
    x = torch.from_numpy(synth.random_flm(L, 0, seed=2, sigma=synth.SIGMA_RED, real=True)).to(dev)
    P = api.Plan(L, 0, sampling=api.HEALPIX, nside=nside, reality=True, device=dev)
    add(f"configs[2] HEALPix nside={nside} L={L} spin-0 real", P, x, pk["dfma"], {"note": "round trip inexact by design"})
    del P, x
    torch.cuda.empty_cache()
    # configs[3]: Wigner transform, L = 256, N = 8
    L, N = 256, 8
    x = torch.from_numpy(synth.random_flmn(L, N, seed=3)).to(dev)
    P = api.Plan(L, N=N, device=dev)
    add(f"configs[3] SO(3) MW L={L} N={N}", P, x, pk["dfma"])
    del P, x
    torch.cuda.empty_cache()
    return rows


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-sweep", action="store_true", help="skip the vs-L sweep of the other configurations")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--L", type=int, default=None, help="profiling only: override the band-limit of the workload")
    ap.add_argument("--spin", type=int, default=None, help="profiling only: override the spin of the workload")
    ap.add_argument("--dtype", default="f64", choices=["f64", "f32"], help="profiling only: fp32 variant (needs --spin 0)")
    ap.add_argument("--shard", default="none", choices=["none", "rings"],
                    help="rings: ONE transform pair per step spread over the --gpus ranks by ring shards (strong scaling; NCCL all-reduce of "
                         "the partial flm and of the map); default: independent problems per rank (weak scaling, no data-path collective)")
    ap.add_argument("--batch", type=int, default=1, help="profiling only: transform a batch of maps together (configs[4]: --L 2048 --spin 0 --batch 16)")
    args = ap.parse_args()
    if args.L is not None:
        WORKLOAD["L"] = args.L
    if args.spin is not None:
        WORKLOAD["spin"] = args.spin
        WORKLOAD["seed"] = 1 if args.spin == 2 else 4
    if args.impl == "reference":
        return run_reference(args)

    import torch
    from paper_2311_14670_b200 import api, synth
    from paper_2311_14670_b200.ranks import Ranks
    from paper_2311_14670_b200.sharded import ShardedTransform

    R = Ranks(backend="nccl")
    rank, local_rank, world = R.rank, R.local_rank, R.world
    torch.cuda.set_device(local_rank)
    dev = torch.device(f"cuda:{local_rank}")
    sync = torch.cuda.synchronize

    L, spin, B = WORKLOAD["L"], WORKLOAD["spin"], args.batch
    sharded = args.shard == "rings"
    # weak scaling (default): every rank transforms its own seeded field (independent problems, no data-path collective);
    # --shard rings: all ranks work on the SAME field, each on its share of the rings (strong scaling)
    if B == 1:
        flm_h = synth.random_flm(L, spin, seed=WORKLOAD["seed"] if sharded else R.seed(WORKLOAD["seed"]), sigma=sigma_for(spin))
    else:
        flm_h = np.stack([synth.random_flm(L, spin, seed=4 + i + 1000 * rank, sigma=synth.SIGMA_RED) for i in range(B)])
    if args.dtype == "f32":
        flm_h = flm_h.astype(np.complex64)
    flm = torch.from_numpy(flm_h).to(dev)
    # (ring shards need the inverse on the MW rings themselves: the midpoint-ring resampling of the default plan mixes rings)
    plan = api.Plan(L, spin, device=dev, batch=B, dtype=args.dtype, invsym=False if sharded else None)
    f = torch.empty(plan.map_shape, dtype=plan.map_dtype, device=dev)
    back = torch.empty_like(flm)
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=dev)      # > 126 MB L2

    if sharded:
        ST = ShardedTransform(plan, R)

        def step():
            ST.inverse(flm, out=f, gather=True)     # each rank fills its rings; the MW forward needs the assembled map
            ST.forward(f, out=back)                 # partial flm of the rank's quadrature rings, summed over ranks
    else:
        def step():
            plan.inverse(flm, out=f)
            plan.forward(f, out=back)

    warm = max(args.warmup, 3)
    for _ in range(warm):
        step()
    R.barrier(sync)
    api.launch_count(reset=True)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    sampler = ClockSampler(local_rank)
    sampler.start()
    R.barrier(sync)
    for a, b in ev:
        flush.zero_()                       # L2 flush between timed iterations (not timed)
        a.record(); step(); b.record()
    R.barrier(sync)
    clocks = sampler.stop()
    launches = api.launch_count()
    total_ms = R.max_over_ranks(sum(a.elapsed_time(b) for a, b in ev), device=dev)
    ms_per_step = total_ms / args.steps
    value = (B * args.steps / (total_ms * 1e-3)) if sharded else R.throughput(B, args.steps, total_ms)
    if sharded:
        plan.set_shard(0, 1)            # the stage timings / e2e / sweep below are single-GPU measurements
    err = float((back - flm).abs().max() / flm.abs().max())

    # per-stage device times: a separate loop of timed transforms AFTER the K timed steps (events recorded inside the library)
    inv_ms, fwd_ms, inv_b, fwd_b, _ = time_stages(plan, flm, flush, reps=5)
    stages = {"inverse_ms": inv_ms, "forward_ms": fwd_ms}

    out = None
    if rank == 0:
        hbm, hbm_kind = peaks()
        pk = {k: api.peak(k, 20000)[0] for k in ("dfma", "dmma", "ffma", "ffma2")}
        nsm = torch.cuda.get_device_properties(dev).multi_processor_count
        peak_tf = pk["ffma"] if args.dtype == "f32" else pk["dfma"]
        # algorithmic flop: per d-step 6 (recursion) + 4 per order and map served
        flops_fwd, flops_inv = plan.flops(True), plan.flops(False)
        fl = flops_fwd / plan.dsteps(True)
        # what the e-form kernels execute per d-step: 2 FP64 instructions of recursion + 2 per order and map served (all FMA-class
        # issue slots): frac_executed = 1.0 means the FP64 pipe issues every cycle (`frac` alone is unbounded by 1)
        orders = (fl - 6.0) / 4.0
        instr = 2.0 + 2.0 * orders
        skf, ski = plan.skip_fraction(True), plan.skip_fraction(False)
        ach = flops_fwd / (stages["forward_ms"]["hot"] * 1e-3) / 1e12
        ach_inv = flops_inv / (stages["inverse_ms"]["hot"] * 1e-3) / 1e12
        kname = ("theta_forward_f32" if args.dtype == "f32" else "theta_forward_kernel" if B == 1 else "theta_mma_kernel<forward>")
        traffic = NCU_TRAFFIC_BYTES.get((L, spin, B)) if args.dtype == "f64" else None
        roof = {"bound": "alu", "kernel": kname + " (fused m-recursion + theta contraction, Eq. 25+30)",
                "achieved": ach, "peak": peak_tf, "unit": "TFLOP/s", "frac": ach / peak_tf,
                "frac_is": "ALGORITHMIC flop (6 per d-step of Eq. 25 as the paper states it + 4 per order served) / hot time / measured peak",
                "frac_executed": ach * (2.0 * instr / fl) / peak_tf * (1.0 - skf),
                "frac_executed_is": f"FP64 instructions the e-form kernel executes ({instr:.0f} per d-step, 2 flop each; the d-steps of the skipped silent "
                                    "heads excluded) / hot time / measured peak: 1.0 = pipe-bound",
                "skipped_dsteps": {"forward": skf, "inverse": ski,
                                   "is": "share of the block-steps the fused kernels skip (tiles near the poles project nothing in their first steps; "
                                         "the state those steps leave is stored at plan time, DESIGN.md section 22); `frac` counts ALL d-steps of the "
                                         "recursion as algorithmic work"},
                "traffic": traffic[0] if traffic else None, "traffic_source": traffic[1] if traffic else None,
                "time_source": "CUDA events recorded inside the library around the hot kernels; median of 5 transforms timed after the K timed steps",
                "peak_kind": f"measured in this run by register-only chains (sht_peak): DFMA {pk['dfma']:.2f}, DMMA {pk['dmma']:.2f}, FFMA {pk['ffma']:.2f}, FFMA2 (packed f32x2) {pk['ffma2']:.2f} "
                             f"TFLOP/s; nominal {nsm} SM x 64 DFMA/clk x 2 x 1.965 GHz = {nsm * 64 * 2 * 1.965e-3:.1f}",
                "flop_per_dstep": fl, "dsteps_per_launch": plan.dsteps(True),
                "inverse_kernel": {"achieved": ach_inv, "frac": ach_inv / peak_tf, "frac_executed": ach_inv * (2.0 * instr / fl) / peak_tf * (1.0 - ski)},
                "hbm_peak_gbs": hbm.get("hbm_gbs"), "hbm_peak_kind": hbm_kind,
                "stage_gbs": {"inverse": {"fft": inv_b["fft"] / (inv_ms["fft"] * 1e-3) / 1e9 if inv_ms["fft"] > 0 else None,
                                          "staging": inv_b["staging"] / (inv_ms["staging"] * 1e-3) / 1e9 if inv_ms["staging"] > 0 else None},
                              "forward": {"fft": fwd_b["fft"] / (fwd_ms["fft"] * 1e-3) / 1e9 if fwd_ms["fft"] > 0 else None,
                                          "staging": fwd_b["staging"] / (fwd_ms["staging"] * 1e-3) / 1e9 if fwd_ms["staging"] > 0 else None}}}
        # end to end through host buffers (pinned), H2D + D2H inside the timed region
        fh = torch.empty(plan.map_shape, dtype=plan.map_dtype).pin_memory()
        ch = torch.from_numpy(flm_h).pin_memory()
        bh = torch.empty(plan.coef_shape, dtype=plan.coef_dtype).pin_memory()

        def pair_host():
            if B == 1 and args.dtype == "f64":          # the C-ABI host-buffer calls copy in and out themselves
                api.s2_inverse_host(ch.numpy(), L, spin, out=fh.numpy()); api.s2_forward_host(fh.numpy(), L, spin, out=bh.numpy())
            else:               # batched plans take device pointers: pinned copies around them, same bytes
                flm.copy_(ch, non_blocking=True); plan.inverse(flm, out=f); fh.copy_(f, non_blocking=True)
                f.copy_(fh, non_blocking=True); plan.forward(f, out=back); bh.copy_(back, non_blocking=True)
                sync()
        for _ in range(2):
            pair_host()
        sync()
        t0 = time.perf_counter()
        ne = max(3, min(args.steps, 10))
        for _ in range(ne):
            pair_host()
        sync()
        te = (time.perf_counter() - t0) / ne
        e2e_err = float(np.abs(bh.numpy() - flm_h).max() / np.abs(flm_h).max())
        del fh, ch, bh
        api.cache_clear()
        nbytes = B * L * (2 * L - 1) * (8 if args.dtype == "f32" else 16)
        e2e = {"value": world * B / te, "unit": UNIT, "h2d_bytes_per_step": 2 * nbytes, "d2h_bytes_per_step": 2 * nbytes,
               "ms_per_step": te * 1e3, "roundtrip_err": e2e_err}
        cpu = None
        if not args.no_cpu:
            t_inv, t_fwd, cores, sample = oracle_sample(L, spin, (flm_h if B == 1 else flm_h[0]).astype(np.complex128), n_cols=32)
            cpu = {"value": 1.0 / (t_inv + t_fwd), "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                   "inverse_s": t_inv, "forward_s": t_fwd}
        out = {"metric": metric_name(L, spin), "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": warm,
               "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "strong" if sharded else "weak", "vs_baseline": None, "dtype": args.dtype,
               "data": "synthetic",
               "config": {"workload": workload_name(L, spin, B), "l2": "flushed between timed iterations (256 MiB memset, untimed)",
                          "parallelism": (f"ring shards x{world}: one transform pair per step, NCCL all-reduce of the map ({f.numel() * f.element_size()} B) and of the "
                                          f"partial flm ({flm.numel() * flm.element_size()} B)" if sharded else f"independent x{world}")},
               "roofline": roof, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": launches, "clocks": clocks,
               "stages": stages, "roundtrip_err": err,
               "paper_context": "S2FFT on 1x A100-40GB: 240 s per MW L=8192 round trip, 430 ms at L=1024 (PAPER.md:737-740, Table 3; other hardware)"}
        if not args.no_sweep and world == 1:
            del plan, f, back, flm
            torch.cuda.empty_cache()
            out["sweep"] = sweep(api, synth, torch, dev, flush, pk)
            out["sweep_is"] = ("per direction: hot / fft / staging ms (median of 3, CUDA events inside the library), frac = algorithmic flop / hot ms / "
                               "measured peak (DFMA unless 'peak' says ffma), GB/s = algorithmic bytes of the stage / its time "
                               f"(HBM peak {hbm.get('hbm_gbs')} GB/s {hbm_kind}); pair_ms = one inverse + forward through the normal call path "
                               "(stage timing off: plans with L <= 512 replay captured CUDA graphs), back to back, no L2 flush")
        print(json.dumps(out))
    R.finish()


if __name__ == "__main__":
    main()
