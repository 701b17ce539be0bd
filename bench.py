#!/usr/bin/env python
"""bench.py -- the hot path of arxiv 2407.09700 (integral-direct J/K Fock build) timed on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg3|cfg2|cfg0|cfg4|cfg1:la,lb,lc,ld:K]
                    [--impl reference] [--no-cpu-baseline] [--per-class FILE]

One "step" = one pass of the whole hot path (Rys roots, recurrences, product + contraction,
digestion, final symmetrisation) over the whole kept quartet list of the workload, i.e. one eri_plan_build_jk call
(cfg4: one eri_plan_jk_grad call; cfg1: one eri_list_plan_digest call).  The plan (S0: pair data, Schwarz bounds,
task lists) depends on geometry, basis and threshold only, is built once before the timed region and its host time
is reported as plan_ms.  Default workload: cfg3, the 32-water / 1856-function J/K build the metric is quoted on.

Prints ONE JSON line (rank 0).  value = unique shell quartets evaluated per second over all ranks (the metric's
"screened ERI quartets/s"); ms_per_step is the metric's "J/K Fock build ms/call"; roofline.frac its "% of FP64 peak".
N > 1: every rank evaluates the units with index % N == rank of the same plan (replicated D and pair data) and the
partial Cartesian J~, K~ are summed with one NCCL all-reduce inside the timed region ("strong" scaling).
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
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2407_09700_b200 import workloads as W  # noqa: E402

METRIC = "screened ERI quartets/s (J/K Fock build)"
NOMINAL_FP64_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12   # SMs x FP64 FMA lanes x 2 x max SM clock


def make_workload(name: str):
    """-> (kind, basis, D, thr, quartets or None, description)"""
    if name == "cfg0":
        b, D, thr = W.cfg0(); return "jk", b, D, thr, None, "cfg0 water dimer, 14 fn, tau=0"
    if name == "cfg2":
        b, D, thr = W.cfg2(); return "jk", b, D, thr, None, "cfg2 8-water DZP-like, 192 fn, tau=1e-13"
    if name == "cfg3":
        b, D, thr = W.cfg3(); return "jk", b, D, thr, None, "cfg3 32-water TZ-like with f, 1856 fn, tau=1e-13"
    if name == "cfg4":
        b, D, thr = W.cfg4(); return "grad", b, D, thr, None, "cfg4 16-water TZ-like, 928 fn, J/K gradient, tau=1e-13"
    if name.startswith("cfg1:"):
        _, cls, K = name.split(":")
        cls = tuple(int(x) for x in cls.split(","))
        b, D, q = W.cfg1_class(cls, int(K))
        return "list", b, D, 0.0, q, f"cfg1 class {cls} K={K}, 1e5 listed quartets"
    raise SystemExit(f"unknown workload {name}")


class ClockSampler(threading.Thread):
    """nvidia-smi clocks / throttle reasons while the timed region runs (B200_PROFILING.md 'clocks line')."""
    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.rows, self._stop_evt = index, [], threading.Event()

    def run(self):
        while not self._stop_evt.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-i", str(self.index)],
                                     capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    self.rows.append([x.strip() for x in out.split(",")])
            except Exception:
                pass
            self._stop_evt.wait(0.2)

    def stop(self) -> dict:
        self._stop_evt.set(); self.join(timeout=6)
        sm = sorted(float(r[0]) for r in self.rows if r and r[0].replace(".", "").isdigit())
        reasons = set()
        for r in self.rows:
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        mx = [float(r[1]) for r in self.rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": mx[0] if mx else None,
                "reasons": sorted(reasons), "samples": len(self.rows)}


def cpu_baseline(kind: str, basis, D, quartets):
    """The oracle as it stands on the host cores, on a bounded sample of the same workload (about 10-30 s)."""
    import oracle
    cores = oracle.num_threads()
    if kind == "list":
        n = max(4, min(len(quartets), 64))
        t = time.perf_counter(); oracle.digest_list(basis, D, quartets[:n]); dt = time.perf_counter() - t
        return {"value": n / dt, "unit": "quartets/s", "cores": cores, "kind": "oracle",
                "sample": f"first {n} listed quartets of the workload (McMurchie-Davidson, no symmetry)", "seconds": dt}
    nw = basis.meta.get("n_water", 2)
    sub_n = min(nw, 2 if basis.meta.get("basis") == "tz" else 4)
    sub = W.subcluster(basis, sub_n) if sub_n < nw else basis
    Ds = np.ascontiguousarray(D[:sub.nao, :sub.nao])
    t = time.perf_counter()
    if kind == "grad":
        sub = W.subcluster(basis, 1) if nw > 1 else basis
        Ds = np.ascontiguousarray(D[:sub.nao, :sub.nao])
        oracle.jk_grad(sub, Ds)
        nq = sub.nshell ** 4
    else:
        _, _, nq = oracle.jk(sub, Ds, 0.0)
    dt = time.perf_counter() - t
    # the oracle walks all ORDERED shell quartets (no symmetry); 8 ordered quartets = 1 unique quartet of the GPU list
    return {"value": nq / 8.0 / dt, "unit": "quartets/s", "cores": cores, "kind": "oracle",
            "sample": f"full unscreened {'gradient' if kind == 'grad' else 'J/K'} of the first {sub.meta.get('n_water', '?')} water(s) of the workload "
                      f"({sub.nshell} shells, {nq} ordered quartets = {nq // 8} unique-quartet equivalents)", "seconds": dt}


def run_reference(args):
    """--impl reference: the oracle timed on the host cores; each step is the bounded sample of cpu_baseline()."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    kind, basis, D, thr, quartets, desc = make_workload(args.workload)
    res = None
    times = []
    for it in range(args.warmup + args.steps):
        res = cpu_baseline(kind, basis, D, quartets)
        if it >= args.warmup:
            times.append(res["seconds"])
    ms = 1e3 * float(np.mean(times))
    value = res["value"] * res["seconds"] / (ms / 1e3)
    cb = dict(res); cb["value"] = value
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": "quartets/s", "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": {"workload": desc, "sample": res["sample"]},
            "cpu_baseline": cb, "e2e": {"value": value, "unit": "quartets/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="cfg3")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--kernel-mode", type=int, default=0, help="0 tuned kernels (default), 1 generic reference kernels")
    ap.add_argument("--per-class", default=None, help="write the per-class table (ms, GFLOP/s, %% of peak) to this file")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import torch
    from paper_2407_09700_b200 import eri   # raises if liberi_b200.so is missing: there is no CPU fallback

    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl")
    kind, basis, D, thr, quartets, desc = make_workload(args.workload)
    nao, natm = basis.nao, basis.natm

    fp64_peak = eri.eri_measure_fp64_peak()
    if kind == "list":
        plan = eri.eri_list_plan_create(basis, quartets)
    else:
        plan = eri.eri_plan_create(basis, thr, want_grad=(kind == "grad"))
    plan.set_kernel_mode(args.kernel_mode)
    if world > 1:
        plan.set_shard(rank, world)
    st = plan.stats()
    Dd = torch.from_numpy(D).cuda()
    J = torch.empty((nao, nao), dtype=torch.float64, device="cuda"); K = torch.empty_like(J)
    gJ = torch.empty((natm, 3), dtype=torch.float64, device="cuda"); gK = torch.empty_like(gJ)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")   # > 126 MB L2

    def step():
        if kind == "grad":
            plan.jk_grad(Dd, gJ, gK)
            if world > 1:
                dist.all_reduce(gJ); dist.all_reduce(gK)
        else:
            plan.build_jk(Dd, J, K)   # N > 1: the library leaves the partial sums; S7 is linear, so reduce the results
            if world > 1:
                dist.all_reduce(J); dist.all_reduce(K)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        flush.fill_(1); step()
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    if sampler:
        sampler.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    for a, b in ev:
        flush.fill_(1)           # L2 flush between timed iterations, outside the event pair
        a.record(); step(); b.record()
    barrier()
    total_ms = sum(a.elapsed_time(b) for a, b in ev)
    clocks = sampler.stop() if sampler else None
    # one more step in timing mode (class launches serialised on one stream, an event between them) for the per-class
    # device times behind `roofline`; the timed steps above run the class launches concurrently on the library's stream pool
    plan.set_timing(True)
    flush.fill_(1); step(); barrier()
    classes = plan.class_stats()
    plan.set_timing(False)
    if world > 1:
        t = torch.tensor([total_ms], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX); total_ms = float(t.item())
    ms = total_ms / args.steps
    nq = st["quartets_kept"]
    flops = st["canonical_flops_grad"] if kind == "grad" else st["canonical_flops"]

    # end to end through the HOST-buffer entry point: pinned host D in, J/K (or the gradient) out, every step
    Dp = torch.from_numpy(D).pin_memory(); Jp = torch.empty((nao, nao), dtype=torch.float64).pin_memory(); Kp = torch.empty_like(Jp).pin_memory()
    gJp = torch.empty((natm, 3), dtype=torch.float64).pin_memory(); gKp = torch.empty_like(gJp).pin_memory()

    def step_host():
        if kind == "grad":
            plan.jk_grad_host(Dp.numpy(), gJp.numpy(), gKp.numpy())
        else:
            plan.build_jk_host(Dp.numpy(), Jp.numpy(), Kp.numpy())

    e2e = None
    if world == 1:
        step_host(); barrier()
        t0 = time.perf_counter()
        n_e2e = max(1, min(args.steps, 3))
        for _ in range(n_e2e):
            step_host()
        barrier()
        e2e_ms = 1e3 * (time.perf_counter() - t0) / n_e2e
        h2d = nao * nao * 8
        d2h = 2 * natm * 3 * 8 if kind == "grad" else 2 * nao * nao * 8
        e2e = {"value": nq / (e2e_ms * 1e-3), "unit": "quartets/s", "ms_per_step": e2e_ms, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h}

    if rank != 0:
        return
    key = "last_ms_grad" if kind == "grad" else "last_ms"
    kern_ms = sum(c[key] for c in classes)
    top = max(classes, key=lambda c: c[key]) if classes else None
    achieved = flops / world / (kern_ms * 1e-3) / 1e12 if kern_ms > 0 else 0.0
    # DRAM traffic of the dominant launch from its `ncu --set full` capture (profiles/r01d_cfg3.md): only known for the launch
    # that was captured, the (dp|dp) K = 1 unit of cfg3 (dram__bytes_read.sum + dram__bytes_write.sum = 48.0 + 137.0 MB)
    traffic = None
    if top is not None and kind == "jk" and args.workload == "cfg3" and [top["la"], top["lb"], top["lc"], top["ld"], top["ka"], top["kb"], top["kc"], top["kd"]] == [2, 1, 2, 1, 1, 1, 1, 1]:
        traffic = 185.0e6
    roofline = {"bound": "alu", "achieved": achieved, "peak": fp64_peak, "unit": "TFLOP/s", "frac": achieved / fp64_peak if fp64_peak else None,
                "traffic": traffic, "traffic_note": "bytes per launch of top_class (ncu --set full, profiles/r01d_cfg3.md); null when that launch was not captured", "peak_source": "FP64 DFMA rate measured in this run (eri_measure_fp64_peak); nominal "
                f"{NOMINAL_FP64_TFLOPS:.1f} = 148 SMs x 64 lanes x 2 x 1.965 GHz", "frac_of_nominal": achieved / NOMINAL_FP64_TFLOPS,
                "kernel": "all class kernels of one step (canonical FLOPs of the kept quartets / summed device time of the class launches, measured in one extra serialised step with an event between launches)",
                "class_kernels_share_of_step": kern_ms / ms if ms else None,
                "top_class": None if top is None else {"l": [top["la"], top["lb"], top["lc"], top["ld"]], "k": [top["ka"], top["kb"], top["kc"], top["kd"]],
                                                       "ms": top[key], "quartets": top["quartets"],
                                                       "tflops": ((top["canonical_flops_grad"] if kind == "grad" else top["canonical_flops"]) / (top[key] * 1e-3) / 1e12) if top[key] > 0 else None}}
    cb = None
    if not args.no_cpu_baseline and world == 1:
        cb = cpu_baseline(kind, basis, D, quartets)
    line = {"metric": METRIC, "value": nq / (ms * 1e-3), "unit": "quartets/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms, "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": desc, "nao": nao, "nshell": basis.nshell, "quartets_kept": nq, "quartets_total": st["quartets_total"],
                       "pairs_kept": st["pairs_kept"], "canonical_flops": flops, "plan_ms": st["plan_ms"], "l2": "flushed between timed steps (256 MB fill)",
                       "kernel_mode": args.kernel_mode, "parallelism": "replicated plan, units dealt round-robin, NCCL all-reduce of J,K" if world > 1 else "single GPU"},
            "jk_build_ms_per_call": ms, "canonical_tflops": flops / (ms * 1e-3) / 1e12, "fp64_peak_measured_tflops": fp64_peak,
            "pct_of_fp64_peak": 100.0 * flops / (ms * 1e-3) / 1e12 / fp64_peak,
            "clocks": clocks, "e2e": e2e, "gpu_launches": (st["launches_per_call"]) * args.steps, "roofline": roofline, "cpu_baseline": cb}
    if args.per_class:
        with open(args.per_class, "w") as f:
            f.write("la lb lc ld ka kb kc kd N kernel quartets ms canonical_GFLOPs TFLOP/s pct_peak unit slots\n")
            for u, c in enumerate(classes):
                c["unit"] = u
            for c in sorted(classes, key=lambda c: -c[key]):
                fl = c["canonical_flops"] if kind != "grad" else c["canonical_flops_grad"]
                tf = fl / (c[key] * 1e-3) / 1e12 if c[key] > 0 else 0.0
                f.write(f"{c['la']} {c['lb']} {c['lc']} {c['ld']} {c['ka']} {c['kb']} {c['kc']} {c['kd']} {c['nroots']} {c['kernel_grad'] if kind == 'grad' else c['kernel']} "
                        f"{c['quartets']} {c[key]:.4f} {fl / 1e9:.3f} {tf:.3f} {100 * tf / fp64_peak:.2f} {c['unit']} {c['slots']}\n")
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
