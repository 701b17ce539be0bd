"""Host-side logic of bench.py (no GPU): the `--gpus N` launcher, the kept-quartet counting behind the projected CPU
baseline, and the compact sub-basis used to time oracle samples."""
import json
import os
import subprocess
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import bench  # noqa: E402
from paper_2407_09700_b200 import workloads as W  # noqa: E402


def test_gpus_2_starts_two_ranks():
    """`python bench.py --gpus 2` with no RANK in the environment re-executes itself under torch.distributed.run with 2 ranks"""
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK")}
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--launch-check"], capture_output=True, text=True,
                         env=env, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads([x for x in out.stdout.splitlines() if x.startswith("{")][-1])
    assert line["n_gpus"] == 2 and len(set(line["pids"])) == 2 and 0 not in line["pids"]


def test_world_size_mismatch_is_refused():
    env = dict(os.environ, RANK="0", WORLD_SIZE="1", LOCAL_RANK="0")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--launch-check"], capture_output=True, text=True,
                         env=env, timeout=120)
    assert out.returncode != 0


def test_kept_counts_match_brute_force(orc):
    basis, D, _ = W.cfg2()
    Q = orc.schwarz(basis)
    thr = 1e-6   # loose enough to screen a lot on the 8-water cluster
    got = bench._kept_counts_per_lclass(basis, Q, thr)
    l = basis.shells["l"]
    iu, ju = np.tril_indices(basis.nshell)
    la, lb = np.maximum(l[iu], l[ju]), np.minimum(l[iu], l[ju])
    q = Q[iu, ju]
    keep = q[:, None] * q[None, :] >= thr
    idx = np.arange(len(q))
    want = {}
    for P in sorted(set(zip(la.tolist(), lb.tolist()))):
        for R in sorted(set(zip(la.tolist(), lb.tolist()))):
            if R > P:
                continue
            mp, mr = (la == P[0]) & (lb == P[1]), (la == R[0]) & (lb == R[1])
            sub = keep[np.ix_(mp, mr)]
            n = int(sub.sum()) if P != R else int(np.triu(sub).sum())   # unordered pairs of pairs incl. the diagonal
            if n:
                want[P + R] = n
    assert got == want
    assert sum(bench._kept_counts_per_lclass(basis, Q, 0.0).values()) == len(q) * (len(q) + 1) // 2


def test_compact_sub_basis_gives_the_same_digest(orc):
    basis, D, _ = W.cfg2()
    rng = np.random.default_rng(3)
    q = rng.integers(0, basis.nshell, (12, 4)).astype(np.int32)
    Jt, Kt = orc.digest_list(basis, D, q)
    sub, Ds, qs = bench._compact(basis, D, q)
    Js, Ks = orc.digest_list(sub, Ds, qs)
    used = np.unique(q)
    ao = np.concatenate([np.arange(basis.shells["ao_off"][s], basis.shells["ao_off"][s] + 2 * basis.shells["l"][s] + 1) for s in used])
    assert np.allclose(Jt[np.ix_(ao, ao)], Js, atol=1e-14) and np.allclose(Kt[np.ix_(ao, ao)], Ks, atol=1e-14)
