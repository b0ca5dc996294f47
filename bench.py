#!/usr/bin/env python
"""bench.py -- (T) FP64 throughput on B200 (BASELINE.json metric), one JSON line on stdout.

A "step" is one pass of the whole hot path over one synthetic
problem: tc_triples_energy with DF-factor input, i.e. triplet scheduling, DF -> integral-block
assembly, the fused W contractions + on-chip epilogue, and the reductions.  Default workload:
BASELINE.json configs[1] (o=20, v=200, naux=600, seed 1), inputs resident in HBM.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config cfg1] [--impl ours|reference]

N > 1 (torchrun): the linear triplet index is partitioned into N contiguous ranges, one per
rank; the only exchange is one all-reduce of the FP64 partial energy.  `value` is whole-job
TFLOP/s = executed contraction flop of all ranks / max-over-ranks device time.

--impl reference times the CPU oracle (oracle/, plain C loops) on the host cores, on a bounded
triplet sample of the same workload.
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

METRIC = "(T) FP64 TFLOP/s (executed o^3v^4 + o^4v^3 contraction flop / E(T) time), 1 GPU"
UNIT = "TFLOP/s"


def flops_per_triplet(o, v):
    return 12.0 * v ** 3 * (v + o)


def nonzero_in_range(o, first, count):
    from paper_2512_01055_b200 import binding
    return sum(1 for n in range(first, first + count) if binding.triplet_decode(o, n)[3] != 0.0)


def partition(ntrip, world, rank):
    """Contiguous range of the linear triplet index owned by `rank` (sizes differ by at most one)."""
    base, rem = divmod(ntrip, world)
    first = rank * base + min(rank, rem)
    return first, base + (1 if rank < rem else 0)


class ClockSampler:
    """nvidia-smi SM clock / throttle reasons during the timed region (B200_PROFILING.md recipe)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "200"], stdout=subprocess.PIPE, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        sm = [float(r[0]) for r in self.rows if r and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        pw = [float(r[2]) for r in self.rows if len(r) > 2 and r[2].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for q, n in enumerate(names) if any(len(r) > 3 + q and r[3 + q] == "Active" for r in self.rows)]
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": reasons}


def oracle_sample(prob_cfg, seconds_target=15.0):
    """Time the CPU oracle on a bounded triplet sample of the workload; returns a cpu_baseline dict."""
    import oracle
    from paper_2512_01055_b200 import synth
    o, v, naux, seed = synth.config_sizes(prob_cfg)
    p = synth.make_config(prob_cfg)
    # the sample: the last triplets of the linear index (all-distinct i>j>k, the common case)
    ntrip = oracle.triplet_count(o)
    first = ntrip - 1
    i, j, k, _ = oracle.triplet_decode(o, first)
    slices = {x: synth.vvvo_slice(p, x) for x in {i, j, k}}
    if p.ovoo is None:
        p.ovoo = np.ascontiguousarray(np.einsum("qlj,qkc->jklc", p.Boo, p.Bov, optimize=True))
        p.ovov = np.ascontiguousarray(np.einsum("qjb,qkc->jkbc", p.Bov, p.Bov, optimize=True))
    t0 = time.perf_counter()
    oracle.triples_energy_slices(p, slices, first, 1)
    t1 = time.perf_counter() - t0
    n = int(max(1, min(64, seconds_target / max(t1, 1e-3))))
    # n consecutive triplets ending at the last index; they share i and mostly j
    first = ntrip - n
    need = set()
    for q in range(first, ntrip):
        need.update(oracle.triplet_decode(o, q)[:3])
    slices = {x: slices[x] if x in slices else synth.vvvo_slice(p, x) for x in need}
    t0 = time.perf_counter()
    oracle.triples_energy_slices(p, slices, first, n)
    dt = time.perf_counter() - t0
    nz = sum(1 for q in range(first, ntrip) if oracle.triplet_decode(o, q)[3] != 0.0)
    return {"value": nz * flops_per_triplet(o, v) / dt * 1e-12, "unit": UNIT, "cores": oracle.num_threads(),
            "kind": "oracle", "sample": f"{n} triplets [{first},{ntrip}) of {prob_cfg}, {dt:.2f} s",
            "seconds_per_triplet": dt / n}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_2512_01055_b200 import synth
    o, v, naux, seed = synth.config_sizes(args.config)
    per_step = []
    cb = None
    for s in range(args.warmup + args.steps):
        cb = oracle_sample(args.config, seconds_target=max(2.0, 60.0 / max(1, args.steps + args.warmup)))
        if s >= args.warmup:
            per_step.append(cb)
    val = float(np.mean([c["value"] for c in per_step]))
    ms = float(np.mean([c["seconds_per_triplet"] for c in per_step])) * 1e3
    cb = dict(per_step[-1], value=val)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"{args.config} (o={o}, v={v}, naux={naux}, seed {seed}); each step = the CPU oracle on a "
                               f"bounded triplet sample; ms_per_step is per triplet"},
        "cpu_baseline": cb,
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2512_01055_b200 import binding, synth

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    torch.cuda.set_device(local)
    ctx = binding.Context(local)
    o, v, naux, seed = synth.config_sizes(args.config)
    ntrip = binding.triplet_count(o)
    first, count = partition(ntrip, world, rank)
    if args.config == "cfg4" and world == 1 and not args.triplets and args.first < 0:
        first, count = 59640, 2000      # BASELINE.json configs[4]: a fixed contiguous slice of 2000 triplets (reading 14)
    if args.first >= 0:
        first = args.first
        count = min(count, ntrip - first)
    if args.triplets:
        count = min(count, args.triplets)

    # ---- inputs: seeded, synthetic, generated on the host, resident in HBM before timing ----
    # (problems whose t2 exceeds 8 GB derive the MP2 amplitudes from the uploaded B_ov on the device)
    big = 8.0 * o * o * v * v > 8e9
    p = synth.make_config(args.config, with_t2=not big)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    names = ("eps_occ", "eps_vir", "t1", "Boo", "Bov", "Bvv") + (() if big else ("t2",))
    if big:
        host = {}
        d = {k: torch.from_numpy(np.ascontiguousarray(getattr(p, k))).cuda() for k in names}
        d["t2"] = synth.mp2_amplitudes_device(d["Bov"], d["eps_occ"], d["eps_vir"])
    else:
        host = {k: pin(getattr(p, k)) for k in names}
        d = {k: t.cuda(non_blocking=True) for k, t in host.items()}
    torch.cuda.synchronize()
    # workspace: everything the library needs; if all (vv|vo) slices do not fit it sizes a slice cache instead
    free_b = torch.cuda.mem_get_info()[0] - (3 << 30)
    nb = ctx.workspace_bytes(o, v, naux, free_b)
    ws = torch.empty(nb, dtype=torch.uint8, device="cuda")
    torch.cuda.synchronize()
    df = (naux, d["Boo"], d["Bov"], d["Bvv"])

    def step():
        return ctx.triples_energy_slice(o, v, d["eps_occ"], d["eps_vir"], d["t1"], d["t2"], df=df, workspace=ws,
                                        workspace_bytes=nb, first=first, count=count)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        E = step()
    sampler = ClockSampler(local)
    barrier()
    if rank == 0:
        sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ms_contr, launches = [], 0
    e0.record()
    for _ in range(args.steps):
        E = step()
        st = ctx.get_stats()
        ms_contr.append(st["ms_contraction"])
        launches += st["n_kernel_launches"]
    e1.record()
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    ms = e0.elapsed_time(e1) / args.steps
    st = ctx.get_stats()
    flop = st["flop_contraction"]
    tmax = torch.tensor([ms], dtype=torch.float64, device="cuda")
    ftot = torch.tensor([flop, E], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
        dist.all_reduce(ftot, op=dist.ReduceOp.SUM)   # whole-job flop and the one scalar the method exchanges: E
    ms_all, flop_all, E_all = float(tmax[0]), float(ftot[0]), float(ftot[1])

    # ---- end to end through the host-pointer C-ABI call (H2D copies inside the timed region) ----
    e2e = None
    if world == 1 and not args.no_e2e and not big:
        hb = [host[k].numpy() for k in ("eps_occ", "eps_vir", "t1", "t2", "Boo", "Bov", "Bvv")]
        del ws
        torch.cuda.empty_cache()
        ctx.triples_energy_host(o, v, naux, *hb, first=first, count=count)   # warm-up
        n_e2e = max(1, min(args.steps, 3))
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            E_h, h2d = ctx.triples_energy_host(o, v, naux, *hb, first=first, count=count)
        dt = (time.perf_counter() - t0) / n_e2e
        e2e = {"value": flop / dt * 1e-12, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": 8,
               "ms_per_step": dt * 1e3, "E": E_h}

    if rank != 0:
        return
    # ---- roofline of the dominant kernel (fused W-builder): FP64 tensor pipe ----
    dmma_sus, dmma_burst = ctx.bench_dmma_peak(2.0)
    ms_k = float(np.mean(ms_contr))
    achieved = flop / (ms_k * 1e-3) * 1e-12
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    # DRAM bytes of one k_wbuild_tma launch from ncu (profiles/r01e_committed_kernel.md): measured on the full cfg1 range
    traffic = 216451098880 + 3586434304 if (args.config == "cfg1" and world == 1 and count == ntrip) else None
    roofline = {"bound": "tensor", "kernel": "k_wbuild_tma", "achieved": achieved, "peak": dmma_sus, "unit": UNIT,
                "frac": achieved / dmma_sus, "traffic": traffic, "traffic_unit": "bytes per launch (dram read+write, ncu)",
                "peak_source": "FP64 DMMA.8x8x4 microbenchmark measured in this run (sustained 2 s); "
                               f"burst {dmma_burst:.2f}; MEASURED_PEAKS.json has no FP64 figure "
                               f"(bf16 {peaks.get('bf16_tflops')} TF/s, hbm {peaks.get('hbm_gbs')} GB/s)",
                "kernel_ms_per_step": ms_k}
    cb = None if args.no_cpu else oracle_sample(args.config)
    out = {
        "metric": METRIC, "value": flop_all / (ms_all * 1e-3) * 1e-12, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_all, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"{args.config}: closed-shell (T), o={o}, v={v}, naux={naux}, seed {seed}, "
                               f"triplets [{first},{first + count}) of {ntrip} per rank-0, DF-factor input (a2 staging inside the step)",
                   "l2": "inputs larger than L2 (vvvo %.2f GB vs 126 MB); no explicit flush" % (o * v ** 3 * 8e-9),
                   "parallelism": f"triplet ranges x{world}"},
        "E_T": E_all, "frac_of_dmma_peak": flop_all / (ms_all * 1e-3) * 1e-12 / (dmma_sus * world),
        "staging": {"ms_per_step": st["ms_staging"], "slices_built_per_step": st["slices_built"]},
        "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline, "cpu_baseline": cb,
    }
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="cfg1")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--triplets", type=int, default=0, help="limit the triplet range per rank (profiling runs)")
    ap.add_argument("--first", type=int, default=-1, help="first triplet of the range (linear index)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
