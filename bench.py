#!/usr/bin/env python
"""bench.py — headline measurement of the hsg hot path (BASELINE.json metric: ns per spin update, OR+HB mix).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c4] [--impl ours|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

One "step" is one pass of the whole hot path over every system of the workload:
hsg_sweep(n_or, n_hb) + hsg_pt_swap (energies + swaps) + hsg_measure (E, m, q(0), q(k_min)).
`value` = step time / ((n_or+n_hb) * R * N) in ns, state resident in HBM (1.6 GB for c4, far larger than L2).
`e2e`   = the same metric over one "execution round" driven through the C ABI from HOST
          buffers: J, H and the start spins are copied from pinned host memory, K steps run with the
          observables of every step read back to the host, and the final spins are read back — all inside
          the timed region; bytes per step = round bytes / K.  The round runs as shards of disorder samples,
          one context and stream each, so that the copies of one shard overlap the sweeps of the others.
`roofline` is for the sweep kernel (the dominant one): algorithmic bytes / CUDA-event time.
`cpu_baseline` = the oracle (oracle/, as it stands) timed on the host cores on a bounded sample.
Rank r of an N-GPU run owns its own D samples (sample_offset = r*D): weak scaling, no data-path collective.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import hsg_inputs  # noqa: E402

METRIC = "ns per spin update (OR+HB mix)"
UNIT = "ns/update"


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def _traffic(workload, kernel):
    """(dram bytes per sweep-kernel launch, where the number comes from) from the committed ncu capture listed in
    profiles/traffic.csv (`workload:kernel,bytes,capture`), or (None, why)."""
    p = os.path.join(ROOT, "profiles", "traffic.csv")
    try:
        for line in open(p):
            if line.startswith(f"{workload}:{kernel},"):
                f = line.strip().split(",")
                return float(f[1]), f"profiles/traffic.csv: {f[2] if len(f) > 2 else 'ncu --set full capture'} (not re-measured in this run)"
    except Exception:
        pass
    return None, "no ncu capture of this workload in profiles/traffic.csv"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 50 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "50"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def _dist():
    rank, world = int(os.environ.get("RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))
    return rank, world, int(os.environ.get("LOCAL_RANK", 0))


# ------------------------------------------------------------------------------------------------ oracle arms
def run_oracle(cfg, temps, steps, warmup, n_systems_cap=64, threads=None, precision=32):
    """Time the oracle as it stands on a bounded sample of the workload: the first sample's systems
    (at most n_systems_cap of them), `steps` full steps after `warmup`.  Returns (ns/update, cores, text)."""
    import oracle
    cores = threads or os.cpu_count() or 1
    O = cfg["n_replicas"]
    T = len(temps)
    while O * T > n_systems_cap and T > 2:
        T //= 2
    tsub = temps[:: len(temps) // T][:T]
    L = cfg["L"]
    J = hsg_inputs.couplings(L, 1, cfg["seed"])
    H = hsg_inputs.gaussian_field(L, 1, cfg["h_r"], cfg["seed"]) if cfg["h_r"] > 0 else None
    sim = oracle.Oracle(L, 1, O, tsub, cfg["seed"], precision=precision, n_threads=cores)
    sim.set_disorder(J, H); sim.init_spins()
    def step():
        sim.sweep(cfg["n_or"], cfg["n_hb"]); sim.pt_swap(); sim.measure()
    for _ in range(warmup):
        step()
    t0 = time.perf_counter()
    for _ in range(steps):
        step()
    dt = time.perf_counter() - t0
    updates = (cfg["n_or"] + cfg["n_hb"]) * O * T * L ** 3 * steps
    text = (f"{steps} steps ({cfg['n_or']} OR + {cfg['n_hb']} HB + PT + measure) of 1 sample x {O} replicas x {T} temperatures, "
            f"L={L}, fp{precision} oracle, {cores} threads over systems")
    return dt / updates * 1e9, cores, text, dt / steps * 1e3


def main_reference(args, cfg, temps):
    rank, world, _ = _dist()
    if rank != 0:
        return
    ns, cores, text, ms = run_oracle(cfg, temps, max(1, args.steps), max(0, min(args.warmup, 1)),
                                     n_systems_cap=args.cpu_systems, threads=args.cpu_threads, precision=args.cpu_precision)
    line = {"impl": "reference", "metric": METRIC, "value": ns, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic", "config": {"workload": args.workload, "note": "oracle on host cores, bounded sample"},
            "cpu_baseline": {"value": ns, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": text},
            "e2e": {"value": ns, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------ GPU arm
def main_ours(args, cfg, temps):
    import torch
    import paper_1204_6192_b200 as hsg

    rank, world, local = _dist()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the hsg hot path has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    L, D, O, T = cfg["L"], cfg["n_samples"], cfg["n_replicas"], len(temps)
    n_or, n_hb = cfg["n_or"], cfg["n_hb"]
    N, R = L ** 3, D * O * T
    off = rank * D                                     # weak scaling: every rank owns its own D samples
    J = hsg_inputs.couplings(L, D, cfg["seed"], off)
    H = hsg_inputs.gaussian_field(L, D, cfg["h_r"], cfg["seed"], off) if cfg["h_r"] > 0 else None

    flags = hsg.HSG_FLAG_FAST_MATH if args.fast_math else 0   # a separately reported VARIANT, never the default
    eng = hsg.hsg_create(L, D, O, temps, cfg["seed"], sample_offset=off, kernel=args.kernel, flags=flags)
    if args.no_fuse_energy:
        eng.set_option(hsg.HSG_OPT_FUSE_ENERGY, 0)
    eng.set_disorder(J, H)
    eng.init_spins()
    f64, i32 = torch.float64, torch.int32
    outs = (eng._new((D, O, T), f64), eng._new((D, O, T, 3), f64), eng._new((D, eng.P, T, 3, 3), f64), eng._new((D, eng.P, T, 3, 3, 2), f64))
    acc = eng._new((D, O, max(T - 1, 0)), i32)
    measure = not args.no_measure

    def step():
        eng.sweep(n_or, n_hb)
        eng.pt_swap(out=acc)
        if measure:
            eng.measure(out=outs)

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    barrier()
    n0 = eng.launch_count(); eng.sweep(n_or, n_hb); sweep_launches_per_call = eng.launch_count() - n0
    kernel = eng.last_sweep_kernel()
    two_phase = kernel == "zmarch" and sweep_launches_per_call == 2 and n_or > 0 and n_hb > 0
    eng.pt_swap(out=acc)
    barrier()

    # ---- the timed region: EXACTLY args.steps steps of the product calls (hsg_sweep(n_or, n_hb), hsg_pt_swap, hsg_measure),
    # bracketed by barrier + synchronize, CUDA events on the engine's stream; repeated, and the MEDIAN region is reported
    def timed_region(K):
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        es = [torch.cuda.Event(enable_timing=True) for _ in range(2 * K)]
        barrier()
        l0 = eng.launch_count()
        ev0.record()
        for k in range(K):
            es[2 * k].record()
            eng.sweep(n_or, n_hb)
            es[2 * k + 1].record()
            eng.pt_swap(out=acc)
            if measure:
                eng.measure(out=outs)
        ev1.record()
        barrier()
        t = [ev0.elapsed_time(ev1), sum(es[2 * k].elapsed_time(es[2 * k + 1]) for k in range(K))]
        if dist is not None:
            tt = torch.tensor(t, device="cuda", dtype=torch.float64)
            dist.all_reduce(tt, op=dist.ReduceOp.MAX)
            t = tt.tolist()
        return t[0], t[1], eng.launch_count() - l0

    first_ms, _, _ = timed_region(args.steps)                  # one untimed-in-the-report region sizes the repeat count
    if args.repeats > 0:
        n_rep = args.repeats
    else:                                                      # at least 5 repeats and at least ~1 s of timed work in total
        n_rep = int(min(50, max(5, np.ceil(1000.0 / max(first_ms, 1e-3)))))
    if dist is not None:
        tt = torch.tensor([n_rep], device="cuda"); dist.all_reduce(tt, op=dist.ReduceOp.MAX); n_rep = int(tt.item())
    sampler = ClockSampler(local) if rank == 0 else None
    if sampler:
        sampler.start()
    regions = [timed_region(args.steps) for _ in range(n_rep)]
    clocks = sampler.stop() if sampler else None
    totals = sorted(r[0] for r in regions)
    total_ms = float(np.median(totals))
    sweep_ms = float(np.median([r[1] for r in regions]))
    launches = regions[0][2]

    # ---- per-launch breakdown (roofline only): at L = 32 / 16 hsg_sweep(n_or, n_hb) is an over-relaxation launch followed by
    # a heat-bath launch; a separate pass makes the same two launches through two calls so that each can be timed
    or_ms = 0.0
    if two_phase:
        K2 = min(args.steps, 20)
        fuse = not args.no_fuse_energy
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(3 * K2)]
        barrier()
        for k in range(K2):
            ev[3 * k].record()
            if fuse:
                eng.set_option(hsg.HSG_OPT_FUSE_ENERGY, 0)         # E and m only in the last launch, as in the single call
            eng.sweep(n_or, 0)
            ev[3 * k + 1].record()
            if fuse:
                eng.set_option(hsg.HSG_OPT_FUSE_ENERGY, 1)
            eng.sweep(0, n_hb)
            ev[3 * k + 2].record()
            eng.pt_swap(out=acc)
            if measure:
                eng.measure(out=outs)
        barrier()
        or_k = float(np.median([ev[3 * k].elapsed_time(ev[3 * k + 1]) for k in range(K2)]))
        hb_k = float(np.median([ev[3 * k + 1].elapsed_time(ev[3 * k + 2]) for k in range(K2)]))
        if dist is not None:
            tt = torch.tensor([or_k, hb_k], device="cuda", dtype=torch.float64)
            dist.all_reduce(tt, op=dist.ReduceOp.MAX)
            or_k, hb_k = tt.tolist()
        or_ms, hb_ms = or_k * args.steps, hb_k * args.steps        # scaled to a region of args.steps steps, like sweep_ms

    # ---- end-to-end round through the C ABI from host buffers (rank-local; max over ranks)
    e2e = None
    if not args.no_e2e:
        S0 = eng.get_spins()
        pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
        J_h, H_h = pin(J), (pin(H) if H is not None else None)
        S_h = torch.empty(S0.shape, dtype=torch.float32).pin_memory(); S_h.copy_(S0); del S0
        out_h = [torch.empty(o.shape, dtype=o.dtype).pin_memory() for o in outs] + [torch.empty(acc.shape, dtype=i32).pin_memory()]
        S_back = torch.empty(S_h.shape, dtype=torch.float32).pin_memory()
        # The round runs as K shards of D/K disorder samples, one hsg context and one CUDA stream each (samples are
        # independent: DESIGN.md §8; sample_offset keeps every random stream that of the global sample), so the H2D
        # and D2H copies of one shard overlap the sweeps of the others.
        K = args.e2e_shards if args.e2e_shards > 0 else (8 if D % 8 == 0 and D >= 16 else 4 if D % 4 == 0 and D >= 8 else 1)
        assert D % K == 0, "--e2e-shards must divide the number of samples"
        Ds = D // K
        shards = []
        for k in range(K):
            st = torch.cuda.Stream()
            with torch.cuda.stream(st):
                e = hsg.hsg_create(L, Ds, O, temps, cfg["seed"], sample_offset=off + k * Ds, stream=st, kernel=args.kernel, flags=flags)
                if args.no_fuse_energy:
                    e.set_option(hsg.HSG_OPT_FUSE_ENERGY, 0)
                sl = slice(k * Ds, (k + 1) * Ds)
                dev = dict(J=e._new(J_h[sl].shape, torch.float32), H=(e._new(J_h[sl].shape, torch.float32) if H_h is not None else None),
                           S=e._new(S_h[sl].shape, torch.float32),
                           outs=(e._new((Ds, O, T), f64), e._new((Ds, O, T, 3), f64), e._new((Ds, e.P, T, 3, 3), f64), e._new((Ds, e.P, T, 3, 3, 2), f64)),
                           acc=e._new((Ds, O, max(T - 1, 0)), i32))
            shards.append((e, st, sl, dev))

        def round_():
            for e, st, sl, dev in shards:
                with torch.cuda.stream(st):
                    dev["J"].copy_(J_h[sl], non_blocking=True)
                    if dev["H"] is not None:
                        dev["H"].copy_(H_h[sl], non_blocking=True)
                    dev["S"].copy_(S_h[sl], non_blocking=True)
                    e.set_disorder(dev["J"], dev["H"]); e.set_spins(dev["S"])
                    for _ in range(args.steps):
                        e.sweep(n_or, n_hb)
                        e.pt_swap(out=dev["acc"])
                        e.measure(out=dev["outs"])
                        for h, d in zip(out_h, list(dev["outs"]) + [dev["acc"]]):
                            h[sl].copy_(d, non_blocking=True)
                    e.get_spins(out=dev["S"])
                    S_back[sl].copy_(dev["S"], non_blocking=True)
        round_()                                            # warm-up round
        barrier()
        t0 = time.perf_counter()
        round_()
        barrier()
        e2e_s = time.perf_counter() - t0
        if dist is not None:
            t = torch.tensor([e2e_s], device="cuda", dtype=torch.float64)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            e2e_s = t.item()
        h2d = (J_h.numel() + (H_h.numel() if H_h is not None else 0) + S_h.numel()) * 4
        d2h = S_back.numel() * 4 + args.steps * sum(h.numel() * h.element_size() for h in out_h)
        e2e = {"value": e2e_s * 1e9 / ((n_or + n_hb) * R * N * args.steps), "unit": UNIT,
               "h2d_bytes_per_step": h2d // args.steps, "d2h_bytes_per_step": d2h // args.steps,
               "what": f"one round of {args.steps} steps: J,H,spins H2D from pinned host + steps with per-step observables D2H + spins D2H; "
                       f"{K} sample shard(s), one context and stream each"}

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    updates_step = (n_or + n_hb) * R * N                       # per rank
    ms_step = total_ms / args.steps
    value = ms_step * 1e6 / updates_step / world               # whole job: all ranks' updates in that time
    ns_sweeps = sweep_ms / args.steps * 1e6 / updates_step / world
    # roofline of the sweep kernel: algorithmic bytes per update:
    # every spin read and written once per sweep (24 B) + J,H once per sweep per sample (24 B / (O*T))
    bytes_per_update = 24.0 + 24.0 / (O * T)
    peak, peak_src = _peaks()
    sweeps_gbs = bytes_per_update * updates_step / (sweep_ms / args.steps * 1e-3) / 1e9      # all sweep launches of a step
    step_gbs = bytes_per_update * updates_step / (total_ms / args.steps * 1e-3) / 1e9       # whole step (what `value` times)
    if two_phase:
        # dominant kernel = the over-relaxation launch (n_or of the n_or + n_hb sweeps of a step), from the split pass
        per_launch_updates = n_or * R * N
        launch_ms = or_ms / args.steps
        kname, tkey = f"zmarch_kernel, over-relaxation launch ({n_or} sweeps)", "zmarch_or"
        share = or_ms / (or_ms + hb_ms) * sweep_ms / total_ms
    else:
        per_launch_updates = updates_step / sweep_launches_per_call
        launch_ms = sweep_ms / args.steps / sweep_launches_per_call
        kname, tkey = f"sweep ({kernel}), {sweep_launches_per_call} launch(es) per step", kernel
        share = sweep_ms / total_ms
    achieved = bytes_per_update * per_launch_updates / (launch_ms * 1e-3) / 1e9
    traffic, traffic_src = _traffic(args.workload, tkey)
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": traffic, "traffic_source": traffic_src, "kernel": kname, "peak_source": peak_src,
                "bytes_per_update": bytes_per_update, "launch_ms": launch_ms, "kernel_share_of_step": share,
                # the metric is the OR+HB mix: the same fraction over ALL sweep launches of a step and over the whole step
                "frac_all_sweeps": sweeps_gbs / peak, "frac_whole_step": step_gbs / peak,
                "all_sweeps": {"achieved": sweeps_gbs, "frac": sweeps_gbs / peak, "ms": sweep_ms / args.steps,
                               "share_of_step": sweep_ms / total_ms,
                               "heat_bath_launch_ms": hb_ms / args.steps if two_phase else None},
                "whole_step": {"achieved": step_gbs, "frac": step_gbs / peak, "ms": total_ms / args.steps}}

    if args.cpu_steps > 0:
        ns_cpu, cores, text, _ = run_oracle(cfg, temps, args.cpu_steps, 1)
    else:
        ns_cpu, cores, text = None, 0, "skipped (--cpu-steps 0)"
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_step, "repeats": n_rep, "timed_region_s": total_ms * 1e-3, "timed_total_s": sum(totals) * 1e-3,
            "value_min": totals[0] / args.steps * 1e6 / updates_step / world, "value_max": totals[-1] / args.steps * 1e6 / updates_step / world,
            "spread": (totals[-1] - totals[0]) / total_ms, "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic",
            "config": {"workload": f"{args.workload}: L={L}, {D} samples x {O} replicas x {T} temperatures per GPU, "
                                   f"{n_or} OR + {n_hb} HB + PT{' + measure' if measure else ''} per step",
                       "L": L, "n_samples_per_gpu": D, "n_replicas": O, "n_temps": T, "n_or": n_or, "n_hb": n_hb,
                       "parallelism": f"samples sharded over {world} GPU(s), no collective", "sweep_kernel": kernel,
                       "arithmetic": "fast-math heat-bath VARIANT (HSG_FLAG_FAST_MATH; not the parity arithmetic)" if args.fast_math
                                     else "reference (bit-exact against the oracle)",
                       "l2": "state (spins) far larger than L2; no flush needed"},
            "ns_per_update_sweeps_only": ns_sweeps, "roofline": roofline,
            "cpu_baseline": {"value": ns_cpu, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": text},
            "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks,
            "paper_context": {"gtx480_ns_per_update_1hb_100or": 0.29, "gtx480_1hb_10or": 0.45, "note": "PAPER.md Table 1, other hardware"}}
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100, help="steps per timed region (SURVEY 8(d): 20 warm-up + 100 timed steps, repeated)")
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--repeats", type=int, default=0, help="timed regions (each exactly --steps steps); the median is reported. 0 = at least 5 and at least ~1 s in total")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c4", choices=sorted(hsg_inputs.CONFIGS))
    ap.add_argument("--kernel", default="auto", choices=["auto", "generic", "zmarch"])
    ap.add_argument("--samples", type=int, default=None, help="override the number of disorder samples per GPU")
    ap.add_argument("--n-or", type=int, default=None, help="override the over-relaxation sweeps per step (OR-only / HB-only timing points)")
    ap.add_argument("--n-hb", type=int, default=None, help="override the heat-bath sweeps per step")
    ap.add_argument("--fast-math", action="store_true", help="time the fast-math heat-bath variant (HSG_FLAG_FAST_MATH) instead of the reference arithmetic")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--e2e-shards", type=int, default=0, help="sample shards (contexts + streams) of the end-to-end round; 0 = 8 or 4 if they divide the samples")
    ap.add_argument("--no-measure", action="store_true")
    ap.add_argument("--no-fuse-energy", action="store_true", help="separate energy reduction kernel instead of the fused final sweep")
    ap.add_argument("--cpu-steps", type=int, default=3, help="oracle steps timed for cpu_baseline")
    ap.add_argument("--cpu-threads", type=int, default=None, help="--impl reference: oracle threads (default: all host cores)")
    ap.add_argument("--cpu-systems", type=int, default=64, help="--impl reference: systems in the bounded sample")
    ap.add_argument("--cpu-precision", type=int, default=32, choices=[32, 64], help="--impl reference: oracle instantiation")
    args = ap.parse_args()
    cfg = dict(hsg_inputs.CONFIGS[args.workload])
    if args.samples is not None:
        cfg["n_samples"] = args.samples
    if args.n_or is not None:
        cfg["n_or"] = args.n_or
    if args.n_hb is not None:
        cfg["n_hb"] = args.n_hb
    if cfg["t_min"] == cfg["t_max"]:
        temps = (cfg["t_min"] * (1.0 + 1e-6 * np.arange(cfg["n_temps"]))).astype(np.float32)
    else:
        temps = hsg_inputs.geometric_ladder(cfg["t_min"], cfg["t_max"], cfg["n_temps"])
    if args.impl == "reference":
        main_reference(args, cfg, temps)
    else:
        main_ours(args, cfg, temps)


if __name__ == "__main__":
    main()
