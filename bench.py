#!/usr/bin/env python
"""bench.py -- headline measurement: spin-s SHT inverse + forward on one B200 (and N independent ranks).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--sweep]

A "step" is one pass of the whole hot path over one synthetic input: an inverse transform (flm -> map) followed by
a forward transform (map -> flm) of BASELINE.json's config[1] (spin-2 complex SHT, MW sampling, L = 1024, fp64).
`value` is transform pairs per second over all ranks with inputs resident in HBM; `e2e` is the same through the
host-buffer C-ABI calls (H2D/D2H inside the timed region).  `roofline` is the fused recursion+contraction kernel of
the forward transform against the FP64 FMA-pipe peak; `cpu_baseline` is the CPU oracle on a bounded sample.
One JSON line on stdout (rank 0).
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

WORKLOAD = dict(L=1024, spin=2, seed=1)
METRIC = "SHT fwd+inv transform pairs per second (MW L=1024 spin-2 fp64, 1 B200)"
UNIT = "transform_pairs/s"
# algorithmic flop per d-step: recursion 6 + projection 4 per order served
# dram__bytes_read.sum + dram__bytes_write.sum of the forward theta kernel, per launch, from the ncu --set full captures in
# profiles/r1_v7_theta_kernels.md; key (L, spin, batch).  Not measurable inside this process: null for other workloads.
NCU_TRAFFIC_BYTES = {(1024, 2, 1): 128.008e6 + 11.222e6, (2048, 0, 1): 1.516876e9 + 155.507e6, (2048, 0, 16): 46.314083e9 + 11.453921e9}


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
        sm, smax, reasons = [], [], set()
        for ln in self.lines:
            c = [x.strip() for x in ln.split(",")]
            if len(c) < 9:
                continue
            try:
                sm.append(float(c[1])); smax.append(float(c[2]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), c[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return dict(sm_mhz=statistics.median(sm) if sm else None, sm_max_mhz=max(smax) if smax else None,
                    reasons=sorted(reasons), samples=len(sm))


def oracle_sample(L, spin, flm, n_cols=12, n_rings=6):
    """Time the CPU oracle (as it stands) on a bounded sample and extrapolate to one inverse + one forward.
    Inverse cost is per ring, forward cost per harmonic order m (both ~uniform across rings; per m ~ (L-|m|))."""
    import oracle as O
    rings = np.linspace(0, L - 1, n_rings).astype(int)
    t0 = time.perf_counter()
    rows = O.s2_inverse_rings(L, spin, O.MW, flm, rings)
    t_inv = (time.perf_counter() - t0) * L / n_rings
    # a band-limited map is not needed for timing: the forward's cost does not depend on the values
    f = np.zeros((L, 2 * L - 1), np.complex128)
    for r, row in zip(rings, rows):
        f[r] = row
    ms = np.unique(np.linspace(-(L - 1), L - 1, n_cols).astype(int))
    t0 = time.perf_counter()
    O.s2_forward_columns(L, spin, O.MW, f, ms)
    dt = time.perf_counter() - t0
    # theta-step cost of a column ~ (L - |m|); DFT + upsampling cost is m-independent: scale by the column count
    t_fwd = dt * (2 * L - 1) / len(ms)
    return t_inv, t_fwd, O.threads(), f"inverse: {n_rings} of {L} rings; forward: {len(ms)} of {2 * L - 1} orders m; extrapolated linearly"


def run_reference(args):
    """--impl reference: the CPU oracle on the same config/metric (bounded sample per step)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_2311_14670_b200 import synth
    L, spin = WORKLOAD["L"], WORKLOAD["spin"]
    flm = synth.random_flm(L, spin, seed=WORKLOAD["seed"], sigma=synth.SIGMA_CMB)
    times = []
    sample = ""
    for i in range(args.warmup + args.steps):
        t_inv, t_fwd, cores, sample = oracle_sample(L, spin, flm, n_cols=8, n_rings=4)
        if i >= args.warmup:
            times.append(t_inv + t_fwd)
    t = float(np.mean(times))
    v = 1.0 / t
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": t * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f80 (long double)",
        "data": "synthetic", "config": {"workload": f"MW L={L} spin={spin} complex, inverse+forward", "l2": "n/a (CPU)"},
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--sweep", action="store_true", help="also time the other configs (MW vs L, SO(3)) into the JSON line")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--L", type=int, default=None, help="profiling only: override the band-limit of the workload")
    ap.add_argument("--spin", type=int, default=None, help="profiling only: override the spin of the workload")
    ap.add_argument("--dtype", default="f64", choices=["f64", "f32"], help="profiling only: fp32 variant (needs --spin 0)")
    ap.add_argument("--batch", type=int, default=1, help="profiling only: transform a batch of maps together (configs[4]: --L 2048 --spin 0 --batch 16)")
    args = ap.parse_args()
    if args.L is not None:
        WORKLOAD["L"] = args.L
    if args.spin is not None:
        WORKLOAD["spin"] = args.spin
    if args.impl == "reference":
        return run_reference(args)

    import torch
    from paper_2311_14670_b200 import api, synth

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    dist = None
    if world > 1:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device(f"cuda:{local_rank}"))
    torch.cuda.set_device(local_rank)
    dev = torch.device(f"cuda:{local_rank}")

    L, spin, B = WORKLOAD["L"], WORKLOAD["spin"], args.batch
    # weak scaling: every rank transforms its own seeded field (independent problems, no data-path collective)
    if B == 1:
        flm_h = synth.random_flm(L, spin, seed=WORKLOAD["seed"] + rank, sigma=synth.SIGMA_CMB)
    else:
        flm_h = np.stack([synth.random_flm(L, spin, seed=4 + i + 1000 * rank, sigma=synth.SIGMA_RED) for i in range(B)])
    if args.dtype == "f32":
        flm_h = flm_h.astype(np.complex64)
    flm = torch.from_numpy(flm_h).to(dev)
    plan = api.Plan(L, spin, device=dev, batch=B, dtype=args.dtype)
    f = torch.empty(plan.map_shape, dtype=plan.map_dtype, device=dev)
    back = torch.empty_like(flm)
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=dev)      # > 126 MB L2

    def step():
        plan.inverse(flm, out=f)
        plan.forward(f, out=back)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    api.launch_count(reset=True)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    sampler = ClockSampler(local_rank)
    sampler.start()
    barrier()
    for a, b in ev:
        flush.zero_()                       # L2 flush between timed iterations (not timed)
        a.record(); step(); b.record()
    barrier()
    clocks = sampler.stop()
    launches = api.launch_count()
    total_ms = sum(a.elapsed_time(b) for a, b in ev)
    if dist is not None:
        t = torch.tensor([total_ms], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = float(t.item())
    ms_per_step = total_ms / args.steps
    value = world * B * args.steps / (total_ms * 1e-3)
    err = float((back - flm).abs().max() / flm.abs().max())

    # per-stage device times (CUDA events recorded inside the library on the launching stream)
    plan.enable_timing(True)
    inv_t, fwd_t = [], []
    for _ in range(5):
        flush.zero_(); plan.inverse(flm, out=f); inv_t.append(plan.timings())
        flush.zero_(); plan.forward(f, out=back); fwd_t.append(plan.timings())
    plan.enable_timing(False)
    med = lambda ts, k: statistics.median(t[k] for t in ts)
    stages = {"inverse_ms": {k: med(inv_t, k) for k in ("hot", "fft", "staging", "total")},
              "forward_ms": {k: med(fwd_t, k) for k in ("hot", "fft", "staging", "total")}}

    out = None
    if rank == 0:
        pk, pk_kind = peaks()
        fp64_tf, _ = api.fp64_peak(20000)
        peak_tf = fp64_tf
        if args.dtype == "f32":       # FP32 FMA pipe: 148 SM x 128 lanes x 2 flop x 1.965 GHz (B200_PROFILING.md unit counts; not in MEASURED_PEAKS.json)
            peak_tf = 148 * 128 * 2 * 1.965e-3
        # algorithmic flop: per d-step 6 (recursion) + 4 per order and map served
        flops_fwd = plan.flops(True)
        flops_inv = plan.flops(False)
        fl = flops_fwd / plan.dsteps(True)
        ach = flops_fwd / (stages["forward_ms"]["hot"] * 1e-3) / 1e12
        roof = {"bound": "alu", "kernel": ("theta_forward_f32" if args.dtype == "f32" else "theta_forward_kernel" if B == 1 else "theta_mma_kernel<forward>") + " (fused m-recursion + theta contraction, Eq. 25+30)",
                "achieved": ach, "peak": peak_tf, "unit": "TFLOP/s", "frac": ach / peak_tf,
                "traffic": NCU_TRAFFIC_BYTES.get((L, spin, B)) if args.dtype == "f64" else None,
                "traffic_source": "profiles/r1_v7_theta_kernels.md (ncu --set full, bytes per launch)",
                "peak_kind": "measured in this run by a register-only DFMA chain (sht_fp64_peak); nominal 148 SM x 64 FMA/clk x 2 x 1.965 GHz = 37.2",
                "flop_per_dstep": fl, "dsteps_per_launch": plan.dsteps(True),
                "inverse_kernel": {"achieved": flops_inv / (stages["inverse_ms"]["hot"] * 1e-3) / 1e12,
                                   "frac": flops_inv / (stages["inverse_ms"]["hot"] * 1e-3) / 1e12 / peak_tf},
                "hbm_peak_gbs": pk.get("hbm_gbs"), "hbm_peak_kind": pk_kind}
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
                torch.cuda.synchronize()
        for _ in range(2):
            pair_host()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        ne = max(3, min(args.steps, 10))
        for _ in range(ne):
            pair_host()
        torch.cuda.synchronize()
        te = (time.perf_counter() - t0) / ne
        fh, ch, bh = fh.numpy(), ch.numpy(), bh.numpy()
        nbytes = B * L * (2 * L - 1) * (8 if args.dtype == "f32" else 16)
        e2e = {"value": world * B / te, "unit": UNIT, "h2d_bytes_per_step": 2 * nbytes, "d2h_bytes_per_step": 2 * nbytes,
               "ms_per_step": te * 1e3, "roundtrip_err": float(np.abs(bh - flm_h).max() / np.abs(flm_h).max())}
        cpu = None
        if not args.no_cpu:
            t_inv, t_fwd, cores, sample = oracle_sample(L, spin, (flm_h if B == 1 else flm_h[0]).astype(np.complex128))
            cpu = {"value": 1.0 / (t_inv + t_fwd), "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                   "inverse_s": t_inv, "forward_s": t_fwd}
        out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
               "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": args.dtype,
               "data": "synthetic",
               "config": {"workload": f"{'BASELINE.json configs[1]' if (L, spin, B) == (1024, 2, 1) else 'override'}: spin-{spin} complex SHT, MW sampling L={L} ({L}x{2 * L - 1}), fp64, "
                                      + (f"batch of {B} maps transformed together, " if B > 1 else "") +
                                      "flm ~ N(0, 1/(l(l+1))) l>=2, inverse + forward per step",
                          "l2": "flushed between timed iterations (256 MiB memset, untimed)", "parallelism": f"independent x{world}"},
               "roofline": roof, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": launches, "clocks": clocks,
               "stages": stages, "roundtrip_err": err,
               "paper_context": "S2FFT on 1x A100-40GB: 430 ms per MW L=1024 transform (PAPER.md:737, Table 3; other hardware)"}
        if args.sweep:
            out["sweep"] = sweep(api, synth, torch, dev, flush, fp64_tf)
        print(json.dumps(out))
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


def sweep(api, synth, torch, dev, flush, fp64_tf):
    """ms (hot / fft / staging) and fraction of FP64 peak vs L for MW spin 0, plus the SO(3) config."""
    rows = []
    for L in (64, 256, 512, 1024, 2048, 4096, 8192):
        flm = torch.from_numpy(synth.random_flm(L, 0, seed=4, sigma=synth.SIGMA_RED)).to(dev)
        P = api.Plan(L, 0, device=dev)
        P.enable_timing(True)
        f = P.inverse(flm); b = P.forward(f)
        ti, tf = [], []
        for _ in range(3):
            flush.zero_(); P.inverse(flm, out=f); ti.append(P.timings())
            flush.zero_(); P.forward(f, out=b); tf.append(P.timings())
        mi = {k: min(t[k] for t in ti) for k in ti[0]}
        mf = {k: min(t[k] for t in tf) for k in tf[0]}
        rows.append({"config": f"MW spin-0 L={L}", "inverse_ms": mi, "forward_ms": mf,
                     "inverse_frac_fp64": P.flops(False) / (mi["hot"] * 1e-3) / 1e12 / fp64_tf,
                     "forward_frac_fp64": P.flops(True) / (mf["hot"] * 1e-3) / 1e12 / fp64_tf,
                     "roundtrip_err": float((b - flm).abs().max() / flm.abs().max())})
        del P, f, b, flm
        torch.cuda.empty_cache()
    # BASELINE.json configs[4], fp32 variant (theta_f32.cu): complex64 arrays, fp32 recursion + contraction
    for L in (2048, 8192):
        flm64 = synth.random_flm(L, 0, seed=4, sigma=synth.SIGMA_RED)
        flm = torch.from_numpy(flm64.astype("complex64")).to(dev)
        P = api.Plan(L, 0, device=dev, dtype="f32")
        P.enable_timing(True)
        f = P.inverse(flm); b = P.forward(f)
        ti, tf = [], []
        for _ in range(3):
            flush.zero_(); P.inverse(flm, out=f); ti.append(P.timings())
            flush.zero_(); P.forward(f, out=b); tf.append(P.timings())
        mi = {k: min(t[k] for t in ti) for k in ti[0]}
        mf = {k: min(t[k] for t in tf) for k in tf[0]}
        rows.append({"config": f"MW spin-0 L={L} fp32", "inverse_ms": mi, "forward_ms": mf,
                     "inverse_tflops_fp32": P.flops(False) / (mi["hot"] * 1e-3) / 1e12, "forward_tflops_fp32": P.flops(True) / (mf["hot"] * 1e-3) / 1e12,
                     "fp32_peak_nominal_tflops": 148 * 128 * 2 * 1.965e-3,
                     "roundtrip_err": float((b - flm).abs().max() / flm.abs().max())})
        del P, f, b, flm
        torch.cuda.empty_cache()
    # BASELINE.json configs[4], second half: 16 maps at L = 2048 transformed together (shared recursion, DMMA contraction)
    L, B = 2048, 16
    import numpy as _np
    flm = torch.from_numpy(_np.stack([synth.random_flm(L, 0, seed=4 + i, sigma=synth.SIGMA_RED) for i in range(B)])).to(dev)
    P = api.Plan(L, 0, device=dev, batch=B)
    P.enable_timing(True)
    f = P.inverse(flm); b = P.forward(f)
    ti, tf = [], []
    for _ in range(3):
        flush.zero_(); P.inverse(flm, out=f); ti.append(P.timings())
        flush.zero_(); P.forward(f, out=b); tf.append(P.timings())
    mi = {k: min(t[k] for t in ti) for k in ti[0]}
    mf = {k: min(t[k] for t in tf) for k in tf[0]}
    rows.append({"config": f"MW spin-0 L={L}, batch of {B} maps (theta_mma_kernel, FP64 DMMA)", "inverse_ms": mi, "forward_ms": mf,
                 "inverse_frac_fp64": P.flops(False) / (mi["hot"] * 1e-3) / 1e12 / fp64_tf,
                 "forward_frac_fp64": P.flops(True) / (mf["hot"] * 1e-3) / 1e12 / fp64_tf,
                 "ms_per_map": {"inverse": mi["total"] / B, "forward": mf["total"] / B},
                 "roundtrip_err": float((b - flm).abs().max() / flm.abs().max())})
    del P, f, b, flm
    torch.cuda.empty_cache()
    # BASELINE.json configs[2]: real spin-0 SHT on HEALPix nside = 1024, L = 2048 (forward of the synthesised map: inexact by design)
    nside, L = 1024, 2048
    flm = torch.from_numpy(synth.random_flm(L, 0, seed=2, sigma=synth.SIGMA_RED, real=True)).to(dev)
    P = api.Plan(L, 0, sampling=api.HEALPIX, nside=nside, reality=True, device=dev)
    P.enable_timing(True)
    f = P.inverse(flm); b = P.forward(f)
    ti, tf = [], []
    for _ in range(3):
        flush.zero_(); P.inverse(flm, out=f); ti.append(P.timings())
        flush.zero_(); P.forward(f, out=b); tf.append(P.timings())
    mi = {k: min(t[k] for t in ti) for k in ti[0]}
    mf = {k: min(t[k] for t in tf) for k in tf[0]}
    rows.append({"config": f"HEALPix nside={nside} L={L} spin-0 real", "inverse_ms": mi, "forward_ms": mf,
                 "inverse_frac_fp64": P.flops(False) / (mi["hot"] * 1e-3) / 1e12 / fp64_tf,
                 "forward_frac_fp64": P.flops(True) / (mf["hot"] * 1e-3) / 1e12 / fp64_tf,
                 "roundtrip_err": float((b - flm).abs().max() / flm.abs().max())})
    del P, f, b, flm
    torch.cuda.empty_cache()
    L, N = 256, 8
    c = torch.from_numpy(synth.random_flmn(L, N, seed=3)).to(dev)
    P = api.Plan(L, N=N, device=dev)
    P.enable_timing(True)
    f = P.inverse(c); b = P.forward(f)
    ti, tf = [], []
    for _ in range(3):
        flush.zero_(); P.inverse(c, out=f); ti.append(P.timings())
        flush.zero_(); P.forward(f, out=b); tf.append(P.timings())
    rows.append({"config": f"SO(3) MW L={L} N={N}", "inverse_ms": {k: min(t[k] for t in ti) for k in ti[0]},
                 "forward_ms": {k: min(t[k] for t in tf) for k in tf[0]},
                 "roundtrip_err": float((b - c).abs().max() / c.abs().max())})
    return rows


if __name__ == "__main__":
    main()
