"""Per-instantiation register / spill / shared-memory table from the `-Xptxas -v` logs of the last build.

    python -m paper_2407_09700_b200.build && python -m paper_2407_09700_b200.ptxas_table > profiles/r02_ptxas_table.md

Every kernel instantiation of liberi_b200.so with its registers per thread, spill bytes, stack frame, static shared
memory and the number of warps per SM that the register file alone allows (65536 registers per SM, allocation in units
of 8 registers per thread, 64 warps at most) -- the north star asks for "registers, occupancy and spills for each class".
Dynamic shared memory is set at launch (the *Traits::SMEM constants in csrc/*.cuh) and does not appear in these logs."""
from __future__ import annotations

import glob
import os
import re
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
LOGS = os.path.join(HERE, "csrc", "build", "*.ptxas.log")
THREADS = {"reg_jk_kernel": lambda a: 128, "tile_jk_kernel": lambda a: 32 * a[4] * a[5], "tile_grad_kernel": lambda a: 32 * a[4],
           "tile_grad_team_kernel": lambda a: 96 * a[4], "coop_jk_kernel": lambda a: 32 * max(4, a[4]), "coop_grad_kernel": lambda a: 32 * a[4]}


def demangle(names):
    out = subprocess.run(["c++filt"] + names, capture_output=True, text=True).stdout.splitlines()
    return [o.replace("(int)", "") for o in out]


def rows():
    recs = []
    for log in sorted(glob.glob(LOGS)):
        txt = open(log).read()
        for m in re.finditer(r"Function properties for (\S+)\n\s+(\d+) bytes stack frame, (\d+) bytes spill stores, (\d+) bytes spill loads\n"
                             r"ptxas info\s+: Used (\d+) registers(?:, used (\d+) barriers)?(?:, (\d+) bytes cumulative stack size)?(?:, (\d+) bytes smem)?", txt):
            recs.append((os.path.basename(log)[:-10], m.group(1), int(m.group(2)), int(m.group(3)), int(m.group(4)), int(m.group(5)),
                         int(m.group(8) or 0)))
    names = demangle([r[1] for r in recs])
    out = []
    for (tu, _, stack, sst, sld, regs, smem), name in zip(recs, names):
        m = re.match(r"void eri::(?:\(anonymous namespace\)::)?(\w+)(?:<([^>]*)>)?", name)
        if not m:
            continue
        kern, args = m.group(1), [int(x) for x in m.group(2).split(",")] if m.group(2) else []
        threads = THREADS.get(kern, lambda a: 0)(args) if args else 0
        regs_alloc = (regs + 7) // 8 * 8
        warps = min(64, 65536 // (regs_alloc * 32))
        if threads:
            wpb = threads // 32
            warps = warps // wpb * wpb
        out.append((kern, args, regs, sst, sld, stack, smem, threads, warps, tu))
    return sorted(out, key=lambda r: (r[0], r[1]))


def main():
    rs = rows()
    print("# Registers, spills and register-limited occupancy of every kernel instantiation (ptxas -v, sm_100a)\n")
    print("Command: `python -m paper_2407_09700_b200.build && python -m paper_2407_09700_b200.ptxas_table > profiles/r02_ptxas_table.md` "
          "(nvcc 12.9, `-gencode arch=compute_100a,code=sm_100a -O3 -lineinfo -Xptxas -v`).\n")
    print("Template arguments: `reg_jk_kernel<la,lb,lc,ld>`, `tile_jk_kernel<la,lb,lc,ld,TQ,BI>`, `coop_jk_kernel<la,lb,lc,ld,TW,NCH>`, "
          "`tile_grad_kernel<la,lb,lc,ld,BI,MODE>`, `tile_grad_team_kernel<la,lb,lc,ld,BI>`, `coop_grad_kernel<la,lb,lc,ld,WARPS,EM>`. "
          "`warps/SM (regs)` = resident warps the register file allows, rounded down to whole blocks (shared memory can lower it).\n")
    nspill = sum(1 for r in rs if r[3] or r[4])
    print(f"{len(rs)} kernels, {nspill} with spill traffic; largest spill: "
          + max(rs, key=lambda r: r[3])[0] + "<" + ",".join(map(str, max(rs, key=lambda r: r[3])[1])) + f"> {max(r[3] for r in rs)} B stores.\n")
    print("| kernel | template arguments | registers | spill stores B | spill loads B | stack B | static smem B | threads/block | warps/SM (regs) | translation unit |")
    print("|---|---|---|---|---|---|---|---|---|---|")
    for kern, args, regs, sst, sld, stack, smem, threads, warps, tu in rs:
        print(f"| {kern} | {','.join(map(str, args))} | {regs} | {sst} | {sld} | {stack} | {smem} | {threads or ''} | {warps} | {tu} |")


if __name__ == "__main__":
    main()
