#!/usr/bin/env python
"""bench.py -- the hot path of arxiv 2407.09700 (integral-direct J/K Fock build) timed on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg3|cfg2|cfg0|cfg4|chain|cfg1:la,lb,lc,ld:K|cfg1:all:K]
                    [--impl reference] [--no-cpu-baseline] [--per-class FILE] [--sweep-out FILE] [--density-screen]

One "step" = one pass of the whole hot path (Rys roots, recurrences, product + contraction,
digestion, final symmetrisation) over the whole kept quartet list of the workload, i.e. one eri_plan_build_jk call
(cfg4: one eri_plan_jk_grad call; cfg1: one eri_list_plan_digest call).  The plan (S0: pair data, Schwarz bounds,
task lists) depends on geometry, basis and threshold only, is built once before the timed region and its host time
is reported as plan_ms (plan_ms_second_plan: the same input planned again, without the one-time code loading of a
process's first plan); the one-shot eri_build_jk (plan + build) is timed once and reported as oneshot_ms.
Default workload: cfg3, the 32-water / 1856-function J/K build the metric is quoted on.

Prints ONE JSON line (rank 0).  value = unique shell quartets evaluated per second over all ranks (the metric's
"screened ERI quartets/s"); ms_per_step is the metric's "J/K Fock build ms/call"; roofline.frac its "% of FP64 peak".
N > 1: every rank evaluates the thread blocks b % N == rank of every class launch of the same plan (replicated D and pair
data) and the partial J, K are summed with one NCCL all-reduce inside the timed region ("strong" scaling).  `--gpus N`
with N > 1 and no RANK in the environment re-executes this script under torch.distributed.run with N ranks.
`--workload cfg1:all:K` sweeps the 120 canonical classes of the microbenchmark (BASELINE.json configs[1]) at contraction
degree K, writes one table row per class to --sweep-out and prints one summary JSON line.
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
PROFILE_FACTS = os.path.join(ROOT, "profiles", "top_kernel_facts.json")   # written from ncu captures, see profiles/README.md


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
    if name == "chain":
        b, D, thr = W.chain(); return "jk", b, D, thr, None, f"synthetic chain (SURVEY 8(f) NEXT-4), {b.natm} atoms, {b.nao} fn, tau=1e-10"
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

    def __init__(self, index: int, period: float = 0.2):
        super().__init__(daemon=True)
        self.index, self.rows, self._stop_evt, self.period = index, [], threading.Event(), period

    def run(self):
        while not self._stop_evt.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-i", str(self.index)],
                                     capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    self.rows.append([x.strip() for x in out.split(",")])
            except Exception:
                pass
            self._stop_evt.wait(self.period)

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


# ---------------------------------------------------------------------------------------------------- CPU baseline
def _kept_counts_per_lclass(basis, Q, thr):
    """Unique kept shell quartets per canonical l-class from a Schwarz matrix Q (reading R7): pairs i >= j, quartets
    (ij) >= (kl), kept iff Q_ij Q_kl >= thr.  Pure counting (sort + searchsorted), no method arithmetic."""
    l = basis.shells["l"]
    iu, ju = np.tril_indices(basis.nshell)
    la, lb = np.maximum(l[iu], l[ju]), np.minimum(l[iu], l[ju])
    q = Q[iu, ju]
    groups = {}
    for key in sorted(set(zip(la.tolist(), lb.tolist()))):
        groups[key] = np.sort(q[(la == key[0]) & (lb == key[1])])
    out = {}
    keys = sorted(groups)
    for P in keys:
        for R in keys:
            if R > P:
                continue
            qb, qk = groups[P], groups[R]
            if thr > 0:
                need = np.where(qb > 0, thr / np.maximum(qb, 1e-300), np.inf)
                cnt = len(qk) - np.searchsorted(qk, need, side="left")   # kets with q >= thr / qb
            else:
                cnt = np.full(len(qb), len(qk))
            tot = int(cnt.sum())
            if P == R:   # unordered pairs of pairs, diagonal included
                diag = int(np.count_nonzero(qb * qb >= thr)) if thr > 0 else len(qb)
                tot = (tot + diag) // 2
            if tot:
                out[P + R] = tot
    return out


def _compact(basis, D, quartets):
    """Sub-basis of the shells a quartet sample touches (re-indexed) and the matching density block; keeps the oracle's
    per-thread nao x nao accumulators small, so the timing is the integral work and not their zero-fill."""
    used = np.unique(quartets)
    remap = -np.ones(basis.nshell, dtype=np.int64); remap[used] = np.arange(len(used))
    sh = basis.shells[used].copy()
    ao_idx, prims, ao = [], [], 0
    for s in sh:
        n = 2 * int(s["l"]) + 1
        ao_idx.extend(range(int(s["ao_off"]), int(s["ao_off"]) + n))
        prims.append(basis.prims[int(s["prim_off"]):int(s["prim_off"]) + int(s["nprim"])])
        s["ao_off"] = ao; ao += n
    off = 0
    for s, p in zip(sh, prims):
        s["prim_off"] = off; off += len(p)
    sub = W.Basis(sh, np.concatenate(prims), basis.coords.copy(), ao, dict(basis.meta))
    ao_idx = np.asarray(ao_idx)
    return sub, np.ascontiguousarray(D[np.ix_(ao_idx, ao_idx)]), remap[quartets].astype(np.int32)


def cpu_baseline_jk_projection(basis, D, thr, budget_s: float = 20.0, seed: int = 97):
    """SURVEY 8(d) "oracle timed beside it" for the large J/K workloads: a seeded sample of KEPT quartets per l-class is
    digested by the oracle (oracle.digest_list, as it stands), the per-class seconds per quartet are multiplied by the
    kept counts of the class and summed: a PROJECTION of the oracle's time for the same kept list, labelled so."""
    import oracle
    cores = oracle.num_threads()
    t0 = time.perf_counter()
    Q = oracle.schwarz(basis)                       # the oracle's own bounds: the reference arm uses no GPU code
    t_q = time.perf_counter() - t0
    kept = _kept_counts_per_lclass(basis, Q, thr)
    l = basis.shells["l"]
    by_l = {x: np.where(l == x)[0] for x in set(l.tolist())}
    rng = np.random.default_rng(seed)
    per_class_budget = budget_s / max(1, len(kept))
    proj_s, sampled, t_sample, detail = 0.0, 0, 0.0, {}
    for cls, count in sorted(kept.items()):
        want, got = 4096, []   # rejection-sample kept quartets of the class
        for _ in range(64):
            i = rng.choice(by_l[cls[0]], want); j = rng.choice(by_l[cls[1]], want)
            k = rng.choice(by_l[cls[2]], want); m = rng.choice(by_l[cls[3]], want)
            ok = Q[i, j] * Q[k, m] >= thr
            got.append(np.stack([i[ok], j[ok], k[ok], m[ok]], axis=1))
            if sum(len(g) for g in got) >= 2048:
                break
        pool = np.concatenate(got)[:2048]
        if len(pool) == 0:
            continue
        n, used, secs = 16, 0, 0.0
        while used < len(pool) and secs < per_class_budget:
            batch = pool[used:used + n]
            sub, Ds, qs = _compact(basis, D, batch)
            t = time.perf_counter(); oracle.digest_list(sub, Ds, qs); dt = time.perf_counter() - t
            secs += dt; used += len(batch); n = min(2 * n, 1024)
        per_q = secs / used
        proj_s += per_q * count; sampled += used; t_sample += secs
        detail["".join("spdfg"[x] for x in cls)] = {"kept": count, "sampled": used, "us_per_quartet": 1e6 * per_q}
    nq = sum(kept.values())
    return {"value": nq / proj_s if proj_s > 0 else None, "unit": "quartets/s", "cores": cores, "kind": "oracle",
            "projection": True,
            "sample": f"PROJECTION: {sampled} seeded kept quartets over {len(detail)} l-classes digested by the oracle "
                      f"(McMurchie-Davidson, {t_sample:.1f} s), per-class s/quartet x kept count of the class "
                      f"({nq} kept unique quartets by the oracle's own Schwarz bounds); full list projected at {proj_s:.0f} s",
            "seconds": t_sample, "schwarz_seconds": t_q, "projected_seconds_full_list": proj_s, "quartets_kept_oracle": nq,
            "per_class": detail}


def cpu_baseline(kind: str, basis, D, thr, quartets):
    """The oracle as it stands on the host cores, on a bounded sample of the same workload (about 10-30 s)."""
    import oracle
    cores = oracle.num_threads()
    if kind == "list":
        n = max(4, min(len(quartets), 64))
        t = time.perf_counter(); oracle.digest_list(basis, D, quartets[:n]); dt = time.perf_counter() - t
        return {"value": n / dt, "unit": "quartets/s", "cores": cores, "kind": "oracle",
                "sample": f"first {n} listed quartets of the workload (McMurchie-Davidson, no symmetry)", "seconds": dt}
    nw = basis.meta.get("n_water", 0)
    if kind == "jk" and basis.nshell > 120:
        return cpu_baseline_jk_projection(basis, D, thr)
    t = time.perf_counter()
    if kind == "grad":
        # the oracle has no per-quartet gradient entry point: full unscreened gradient of the first molecule
        sub = W.subcluster(basis, 1) if nw > 1 else basis
        Ds = np.ascontiguousarray(D[:sub.nao, :sub.nao])
        oracle.jk_grad(sub, Ds)
        nq = sub.nshell ** 4
        what = f"full unscreened gradient of the first water of the workload ({sub.nshell} shells)"
    else:
        _, _, nq = oracle.jk(basis, D, 0.0)
        what = f"full unscreened J/K of the workload ({basis.nshell} shells)"
    dt = time.perf_counter() - t
    # the oracle walks all ORDERED shell quartets (no symmetry); 8 ordered quartets = 1 unique quartet of the GPU list
    return {"value": nq / 8.0 / dt, "unit": "quartets/s", "cores": cores, "kind": "oracle",
            "sample": f"{what}: {nq} ordered quartets = {nq // 8} unique-quartet equivalents", "seconds": dt}


def run_reference(args):
    """--impl reference: the oracle timed on the host cores; each step is the bounded sample of cpu_baseline()."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    if args.workload.startswith("cfg1:all"):
        raise SystemExit("--impl reference: name one class, cfg1:la,lb,lc,ld:K")
    kind, basis, D, thr, quartets, desc = make_workload(args.workload)
    res, times = None, []
    for it in range(args.warmup + args.steps):
        res = cpu_baseline(kind, basis, D, thr, quartets)
        if it >= args.warmup:
            times.append(res["seconds"])
    ms = 1e3 * float(np.mean(times))
    cb = {k: v for k, v in res.items() if k != "per_class"}
    line = {"impl": "reference", "metric": METRIC, "value": res["value"], "unit": "quartets/s", "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": {"workload": desc, "sample": res["sample"]},
            "cpu_baseline": cb, "e2e": {"value": res["value"], "unit": "quartets/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# ---------------------------------------------------------------------------------------------------- helpers
def measure_fp64_peak(eri, local: int):
    """FP64 DFMA rate (eri_measure_fp64_peak: 1e5 iterations of 16 independent chains per thread, best of 5) with the SM
    clock sampled while the loop runs."""
    sampler = ClockSampler(local, period=0.05); sampler.start()
    best, t0 = 0.0, time.perf_counter()
    while True:
        best = max(best, eri.eri_measure_fp64_peak())
        if time.perf_counter() - t0 > 1.0:
            break
    clk = sampler.stop()
    return best, clk


def profile_facts(workload: str):
    """Facts about the dominant kernel that only a profiler sees (DRAM bytes per launch, executed FP64 over canonical FLOPs),
    read from the committed ncu summary together with the commit they were captured at; None if there is no capture."""
    try:
        with open(PROFILE_FACTS) as f:
            return json.load(f).get(workload)
    except (OSError, ValueError):
        return None


def self_launch(args) -> int:
    """`--gpus N` (N > 1) outside a launcher: start N ranks of this script under torch.distributed.run on this node."""
    port = 29500 + (os.getpid() % 2000)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    env = dict(os.environ); env.setdefault("NCCL_DEBUG", "WARN")
    return subprocess.call(cmd, env=env)


def launch_check(args):
    """--launch-check: every rank joins a gloo group, the ranks are counted with an all-reduce and rank 0 prints what ran.
    No GPU is touched: this is what the CPU test of the `--gpus N` launcher runs."""
    import torch
    import torch.distributed as dist
    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    if world > 1:
        dist.init_process_group("gloo")
    t = torch.ones(1, dtype=torch.int64)
    pids = torch.zeros(max(world, 1), dtype=torch.int64); pids[rank] = os.getpid()
    if world > 1:
        dist.all_reduce(t); dist.all_reduce(pids)
    assert int(t.item()) == world == args.gpus, (int(t.item()), world, args.gpus)
    if rank == 0:
        print(json.dumps({"launch_check": True, "n_gpus": int(t.item()), "pids": pids.tolist()}))
    if world > 1:
        dist.destroy_process_group()


def sweep_cfg1(args, eri, torch, fp64_peak):
    """cfg1 microbenchmark over all 120 canonical classes at one contraction degree (BASELINE.json configs[1])."""
    K = int(args.workload.split(":")[2])
    classes = W.canonical_classes(4)
    if args.sweep_classes:
        lo, hi = (int(x) for x in args.sweep_classes.split(":"))
        classes = classes[lo:hi]
    rows, tot_flops, tot_ms, launches = [], 0.0, 0.0, 0
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    for cls in classes:
        # the heaviest lists may be shortened so that the K = 6 sweep stays within a gpurun call; the table says so
        nq = 100_000
        if args.sweep_budget_gflop > 0:
            per_q = eri.eri_canonical_flops(*cls, K, K, K, K)
            nq = int(min(100_000, max(2_000, args.sweep_budget_gflop * 1e9 / per_q)))
        basis, D, q = W.cfg1_class(cls, K, nquartets=nq)
        plan = eri.eri_list_plan_create(basis, q)
        st = plan.stats()
        Dd = torch.from_numpy(D).cuda()
        J = torch.empty((basis.nao, basis.nao), dtype=torch.float64, device="cuda"); Kt = torch.empty_like(J)
        for _ in range(max(1, args.warmup)):
            plan.build_jk(Dd, J, Kt)
        torch.cuda.synchronize()
        best = []
        for _ in range(args.steps):
            flush.fill_(1)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); plan.build_jk(Dd, J, Kt); b.record(); torch.cuda.synchronize()
            best.append(a.elapsed_time(b))
        ms = float(np.median(best))
        finite = bool(torch.isfinite(J).all().item() and torch.isfinite(Kt).all().item())
        kinds = sorted({c["kernel"] for c in plan.class_stats()})
        tf = st["canonical_flops"] / (ms * 1e-3) / 1e12
        rows.append((cls, K, nq, ms, nq / (ms * 1e-3), tf, 100.0 * tf / fp64_peak, kinds, finite))
        tot_flops += st["canonical_flops"]; tot_ms += ms; launches += st["launches_per_call"] * args.steps
        plan.destroy()
    if args.sweep_out:
        with open(args.sweep_out, "w") as f:
            f.write("class la lb lc ld K quartets ms quartets_per_s canonical_TFLOPs pct_of_measured_fp64_peak kernel_family finite\n")
            for cls, k, nq, ms, qps, tf, pct, kinds, finite in rows:
                name = "(" + "".join("spdfg"[x] for x in cls[:2]) + "|" + "".join("spdfg"[x] for x in cls[2:]) + ")"
                f.write(f"{name} {cls[0]} {cls[1]} {cls[2]} {cls[3]} {k} {nq} {ms:.4f} {qps:.4e} {tf:.3f} {pct:.2f} {','.join(map(str, kinds))} {int(finite)}\n")
    return rows, tot_flops, tot_ms, launches


def density_screen_lines(plan, Dd, J, K, flush, torch, nq):
    """SURVEY 8(f) NEXT-1 (Eq. 8-9): the same build with the density factor in the screening test, for the
    full density and for an "SCF-like" small change of it (incremental build from delta-D)."""
    out = {}
    gen = torch.Generator(device="cuda"); gen.manual_seed(5)
    dD = torch.randn(Dd.shape, dtype=torch.float64, device="cuda", generator=gen)
    dD = (1e-4 * Dd.abs().max() * 0.5 * (dD + dD.T)).contiguous()
    for name, M in (("D", Dd), ("deltaD_1e-4", dD)):
        for _ in range(2):
            plan.build_jk_dens(M, J, K)
        torch.cuda.synchronize()
        ts = []
        for _ in range(3):
            flush.fill_(1)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); plan.build_jk_dens(M, J, K); b.record(); torch.cuda.synchronize()
            ts.append(a.elapsed_time(b))
        kept = plan.dens_quartets()
        out[name] = {"ms": float(np.median(ts)), "quartets_evaluated": kept, "of_schwarz_kept": kept / nq if nq else None}
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="cfg3")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--kernel-mode", type=int, default=0, help="0 tuned kernels (default), 1 generic reference kernels, 2 no tile family")
    ap.add_argument("--per-class", default=None, help="write the per-unit table (ms, GFLOP/s, %% of peak) to this file")
    ap.add_argument("--sweep-out", default=None, help="cfg1:all:K: write the per-class table to this file")
    ap.add_argument("--sweep-classes", default=None, help="cfg1:all:K: slice lo:hi of the 120 canonical classes")
    ap.add_argument("--sweep-budget-gflop", type=float, default=0.0, help="cfg1:all:K: shorten lists above this many canonical GFLOP (0: always 1e5 quartets)")
    ap.add_argument("--density-screen", action="store_true", help="SURVEY 8(f) NEXT-1: also time the density-weighted build (Eq. 8-9) for D and for a small delta-D")
    ap.add_argument("--launch-check", action="store_true", help="only start the ranks and count them (CPU, gloo)")
    args = ap.parse_args()
    if args.gpus > 1 and "RANK" not in os.environ:
        sys.exit(self_launch(args))
    if args.launch_check:
        return launch_check(args)
    if args.impl == "reference":
        return run_reference(args)

    import torch
    from paper_2407_09700_b200 import eri   # raises if liberi_b200.so is missing: there is no CPU fallback

    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus:
        raise SystemExit(f"--gpus {args.gpus} but WORLD_SIZE = {world}: launch with torch.distributed.run --nproc-per-node {args.gpus}, or without a launcher")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl")
    fp64_peak, peak_clocks = measure_fp64_peak(eri, local)

    if args.workload.startswith("cfg1:all"):
        rows, tot_flops, tot_ms, launches = sweep_cfg1(args, eri, torch, fp64_peak)
        tf = tot_flops / (tot_ms * 1e-3) / 1e12
        line = {"metric": "cfg1 class microbenchmark, canonical TFLOP/s over the swept classes", "value": tf, "unit": "TFLOP/s", "n_gpus": 1,
                "steps": args.steps, "warmup": args.warmup, "ms_per_step": tot_ms, "higher_is_better": True, "scaling": "strong",
                "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": {"workload": args.workload, "classes": len(rows), "table": args.sweep_out,
                           "l2": "flushed between timed calls (256 MB fill)", "shortened_lists": sum(1 for r in rows if r[2] < 100_000)},
                "fp64_peak_measured_tflops": fp64_peak, "fp64_peak_clocks": peak_clocks, "pct_of_fp64_peak": 100.0 * tf / fp64_peak,
                "gpu_launches": launches, "all_finite": all(r[8] for r in rows),
                "worst": min(({"class": r[0], "pct": r[6]} for r in rows), key=lambda x: x["pct"]),
                "best": max(({"class": r[0], "pct": r[6]} for r in rows), key=lambda x: x["pct"])}
        print(json.dumps(line))
        return

    kind, basis, D, thr, quartets, desc = make_workload(args.workload)
    nao, natm = basis.nao, basis.natm
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

    e2e, oneshot_ms, plan_warm = None, None, None
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
        if kind != "list":   # a second plan of the same input: the first one of a process also pays for loading the library's code
            p2 = eri.eri_plan_create(basis, thr, want_grad=(kind == "grad"))
            s2 = p2.stats(); p2.destroy()
            plan_warm = {"plan_ms": s2["plan_ms"], "parts": {k: s2["plan_ms_" + k] for k in ("init", "schwarz", "pairs", "units")}}
        if kind != "list":   # the one-shot call of the north star: plan + build + destroy
            barrier(); t0 = time.perf_counter()
            if kind == "grad":
                eri.eri_jk_grad(basis, Dd, thr)
            else:
                eri.eri_build_jk(basis, Dd, thr)
            barrier(); oneshot_ms = 1e3 * (time.perf_counter() - t0)

    dens = None
    if args.density_screen and kind == "jk" and world == 1:
        dens = density_screen_lines(plan, Dd, J, K, flush, torch, nq)

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return
    key = "last_ms_grad" if kind == "grad" else "last_ms"
    kern_ms = sum(c[key] for c in classes)
    top = max(classes, key=lambda c: c[key]) if classes else None
    achieved = flops / world / (kern_ms * 1e-3) / 1e12 if kern_ms > 0 else 0.0
    facts = profile_facts(args.workload) or {}
    note = ("dram__bytes_read.sum + dram__bytes_write.sum per launch of traffic_kernel, from the committed ncu capture "
            f"{facts.get('source')} taken at commit {facts.get('commit')}") if facts else "no committed ncu capture for this workload"
    roofline = {"bound": "alu", "achieved": achieved, "peak": fp64_peak, "unit": "TFLOP/s", "frac": achieved / fp64_peak if fp64_peak else None,
                "traffic": facts.get("traffic_bytes_per_launch"), "traffic_note": note, "traffic_kernel": facts.get("kernel"),
                "executed_fp64_over_canonical": facts.get("executed_fp64_over_canonical"),
                "peak_source": "FP64 DFMA rate measured in this run (eri_measure_fp64_peak, 1e5 iterations x 16 chains, SM clock sampled: fp64_peak_clocks); nominal "
                f"{NOMINAL_FP64_TFLOPS:.1f} = 148 SMs x 64 lanes x 2 x 1.965 GHz", "frac_of_nominal": achieved / NOMINAL_FP64_TFLOPS,
                "kernel": "all class kernels of one step (canonical FLOPs of the kept quartets / summed device time of the class launches, measured in one extra serialised step with an event between launches)",
                "class_kernels_share_of_step": kern_ms / ms if ms else None,
                "top_class": None if top is None else {"l": [top["la"], top["lb"], top["lc"], top["ld"]], "k": [top["ka"], top["kb"], top["kc"], top["kd"]],
                                                       "ms": top[key], "quartets": top["quartets"],
                                                       "tflops": ((top["canonical_flops_grad"] if kind == "grad" else top["canonical_flops"]) / (top[key] * 1e-3) / 1e12) if top[key] > 0 else None}}
    cb = None
    if not args.no_cpu_baseline and world == 1:
        cb = cpu_baseline(kind, basis, D, thr, quartets)
        cb.pop("per_class", None)
    line = {"metric": METRIC, "value": nq / (ms * 1e-3), "unit": "quartets/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms, "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": desc, "nao": nao, "nshell": basis.nshell, "quartets_kept": nq, "quartets_total": st["quartets_total"],
                       "pairs_kept": st["pairs_kept"], "canonical_flops": flops, "plan_ms": st["plan_ms"],
                       "plan_ms_parts": {k: st["plan_ms_" + k] for k in ("init", "schwarz", "pairs", "units")}, "plan_ms_second_plan": plan_warm, "oneshot_ms": oneshot_ms,
                       "l2": "flushed between timed steps (256 MB fill)", "kernel_mode": args.kernel_mode,
                       "parallelism": f"replicated plan, thread blocks dealt round-robin over {world} ranks, NCCL all-reduce of J,K" if world > 1 else "single GPU"},
            "jk_build_ms_per_call": ms, "canonical_tflops": flops / (ms * 1e-3) / 1e12, "fp64_peak_measured_tflops": fp64_peak,
            "fp64_peak_clocks": peak_clocks, "pct_of_fp64_peak": 100.0 * flops / (ms * 1e-3) / 1e12 / fp64_peak,
            "clocks": clocks, "e2e": e2e, "gpu_launches": (st["launches_per_call"]) * args.steps, "roofline": roofline, "cpu_baseline": cb}
    if dens is not None:
        line["density_screen"] = dens
    if args.per_class:
        with open(args.per_class, "w") as f:
            f.write("la lb lc ld ka kb kc kd N kernel quartets ms canonical_GFLOPs TFLOP/s pct_peak unit slots tile_fill\n")
            for u, c in enumerate(classes):
                c["unit"] = u
            for c in sorted(classes, key=lambda c: -c[key]):
                fl = c["canonical_flops"] if kind != "grad" else c["canonical_flops_grad"]
                tf = fl / (c[key] * 1e-3) / 1e12 if c[key] > 0 else 0.0
                f.write(f"{c['la']} {c['lb']} {c['lc']} {c['ld']} {c['ka']} {c['kb']} {c['kc']} {c['kd']} {c['nroots']} {c['kernel_grad'] if kind == 'grad' else c['kernel']} "
                        f"{c['quartets']} {c[key]:.4f} {fl / 1e9:.3f} {tf:.3f} {100 * tf / fp64_peak:.2f} {c['unit']} {c['slots']} {c['tile_fill_pm'] / 1000:.3f}\n")
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
