"""Writes tests/golden/fullsize_<config>[_call<k>].json: WHOLE-SYSTEM oracle results of a BASELINE.json
config at full size, for the GPU parity tests (tests/test_gpu_parity.py::test_full_size_*).

    python tests/golden/make_fullsize_golden.py --config 3 [--procs P] [--call 99] [--search cells|brute]

Imports only oracle/ and workloads/ -- no value in the output comes from the CUDA path.

What it computes (SURVEY.md 8(d) "Oracle timing" / BASELINE.md section 2: sharded by central-atom range over
host processes, partial forces summed):
  * every centre of the system through oracle.centres(): E_i, the forces of every centre added up (= total
    force on every atom), the neighbour row of every atom;
  * E_total = exactly rounded sum of all E_i (math.fsum), and per SHARD (256 contiguous atom-index ranges):
    sum E_i, sum F, number of neighbour entries and an order-independent 64-bit hash of the (i, j) pairs --
    the whole neighbour list of 2.1 M atoms is compared bit-exactly through these hashes;
  * four seeded random projections sum_m F_m . q_m of the whole force field, sum_m F_m, the histogram of the
    neighbour counts;
  * for >= 64 STRATIFIED atoms: neighbour row, E_i, G_i (from a second run of exactly those centres with the
    BRUTE-FORCE scan, the definition) and F (from the whole-system sum).  Strata: largest / smallest
    neighbour counts, most screening-mask words (the CUDA force kernel's hand-over budget of 320 words per
    centre), first / last cell of each dimension, extreme coordinates, first and last atom of each element in
    (element, cell, index) order, the closest pairs (1/r factors), random fill.

Neighbour search: --search cells (default) uses the oracle's cell-prefiltered scan, which applies the same
predicate to a candidate list and is pinned equal to the brute-force scan (tests/test_oracle_cells_pins.py);
the brute-force scan costs 25 ms per centre at 2.1 M atoms (15 core-hours for configs[3]).  While it runs, the
script re-checks the rows of the stratified atoms and of --check-brute random atoms against the brute-force
scan and records which.
"""
from __future__ import annotations

import argparse
import json
import math
import multiprocessing as mp
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import oracle  # noqa: E402
import workloads as W  # noqa: E402
from workloads import rng  # noqa: E402

HERE = os.path.dirname(os.path.abspath(__file__))
N_SHARDS = 256
PAIR_HASH_KEY = rng.stream_key(2002_00054, 0x6E6272)       # "nbr"
DIGEST_SEED = 2002_00054


def pair_hash(i: np.ndarray, j: np.ndarray) -> int:
    """Order-independent 64-bit digest of a set of ordered pairs: sum over pairs of a 64-bit mix of
    (i << 32 | j), modulo 2^64 (workloads.rng.bits is a bijective mixer of the counter)."""
    c = (i.astype(np.uint64) << np.uint64(32)) | j.astype(np.uint64)
    h = rng.bits(PAIR_HASH_KEY, c)
    with np.errstate(over="ignore"):
        return int(np.add.reduce(h, dtype=np.uint64))


def digest_vectors(n: int, k: int) -> np.ndarray:
    return rng.normal(rng.stream_key(DIGEST_SEED, 0x646967, k), np.arange(3 * n, dtype=np.uint64)).reshape(n, 3)


def system_of(cfg_index: int, call: int):
    cfg = W.CONFIGS[cfg_index]
    sysm, model = W.build(cfg)
    pos = sysm.pos.copy()
    for c in range(1, call + 1):                     # reading C15: cumulative kicks before call c >= 1
        pos = pos + W.displacement(sysm.n_atoms, cfg.seed_disp, c)
    return cfg, sysm, model, pos


def shard_bounds(n: int):
    return [(n * s) // N_SHARDS for s in range(N_SHARDS + 1)]


# ---------------------------------------------------------------------------------- workers
_G = {}


def _worker(wid, cfg_index, call, search, tasks, results, out_dir):
    cfg, sysm, model, pos = system_of(cfg_index, call)
    om = oracle.OracleModel(model)
    n = sysm.n_atoms
    F = np.zeros((n, 3), dtype=np.float64)
    types = sysm.types
    while True:
        t = tasks.get()
        if t is None:
            break
        s, lo, hi = t
        e_atom = np.empty(hi - lo)
        cnt = np.empty(hi - lo, dtype=np.int32)
        cnt0 = np.empty(hi - lo, dtype=np.int32)      # neighbours of element 0 (for the mask-word stratum)
        h, npairs = 0, 0
        t_nbr = t_rest = 0.0
        for a in range(lo, hi, 2048):
            b = min(a + 2048, hi)
            sel = np.arange(a, b, dtype=np.int64)
            r = oracle.centres(om, pos, types, sysm.box, sel, forces=True, want_g=False, search=search, rows=True,
                               F_accum=F)
            e_atom[a - lo:b - lo] = r.e_atom
            cnt[a - lo:b - lo] = r.nbr_count
            owner = np.repeat(sel, np.diff(r.row_off))
            h = (h + pair_hash(owner, r.row_idx)) & ((1 << 64) - 1)
            npairs += int(r.row_off[-1])
            is0 = (types[r.row_idx] == 0).astype(np.int64)
            c0 = np.concatenate([[0], np.cumsum(is0)])
            cnt0[a - lo:b - lo] = c0[r.row_off[1:]] - c0[r.row_off[:-1]]
            t_nbr += r.timing[0]; t_rest += r.timing[1]
        results.put((s, lo, hi, e_atom, cnt, cnt0, h, npairs, t_nbr, t_rest))
    np.save(os.path.join(out_dir, "F_worker_%d.npy" % wid), F)
    results.put(("done", wid))


def mask_words(n0: np.ndarray, n1: np.ndarray) -> np.ndarray:
    """Mask words of the CUDA kernels' screening stream for a two-element centre with n0 / n1 neighbours of
    element 0 / 1 (only used to PICK atoms, never compared)."""
    w = lambda nk: (nk + 31) // 32
    return n0 * w(n0 // 2) + n0 * w(n1) * (n0 > 0) + n1 * w(n1 // 2)


def stratify(pos, types, box, rc, cnt, cnt0, n_random, seed):
    n = pos.shape[0]
    w = oracle.wrap(pos, box)
    nc = np.maximum(np.floor(box / rc).astype(np.int64), 1)
    cell3 = np.minimum((w / box * nc).astype(np.int64), nc - 1)
    cell = (cell3[:, 2] * nc[1] + cell3[:, 1]) * nc[0] + cell3[:, 0]
    picks = {}

    def add(i, why):
        picks.setdefault(int(i), why)

    order = np.argsort(cnt, kind="stable")
    for i in order[::-1][:4]:
        add(i, "largest neighbour count (%d)" % cnt[i])
    for i in order[:2]:
        add(i, "smallest neighbour count (%d)" % cnt[i])
    mw = mask_words(cnt0.astype(np.int64), (cnt - cnt0).astype(np.int64))
    for i in np.argsort(mw, kind="stable")[::-1][:4]:
        add(i, "most screening-mask words (%d; hand-over budget 320)" % mw[i])
    for d in range(3):
        for e in range(int(types.max()) + 1):
            for c, nm in ((0, "first"), (nc[d] - 1, "last")):
                idx = np.flatnonzero((cell3[:, d] == c) & (types == e))
                if idx.size:
                    add(idx[len(idx) // 2], "%s cell of dimension %d, element %d" % (nm, d, e))
        add(np.argmin(w[:, d]), "smallest wrapped coordinate %d" % d)
        add(np.argmax(w[:, d]), "largest wrapped coordinate %d" % d)
    key = np.lexsort((np.arange(n), cell, types))     # (element, cell, original index): the CUDA path's sorted order
    for e in range(int(types.max()) + 1):
        ke = key[types[key] == e]
        add(ke[0], "first atom of element %d in (element, cell, index) order" % e)
        add(ke[-1], "last atom of element %d in (element, cell, index) order" % e)
    # closest pairs (same-element atoms may be arbitrarily close, reading C14): 1/r factors
    from scipy.spatial import cKDTree
    ww = np.where(w >= box, 0.0, w)
    d2, _ = cKDTree(ww, boxsize=box).query(ww, k=2)
    for i in np.argsort(d2[:, 1])[:4]:
        add(i, "closest neighbour at %.5f A" % d2[i, 1])
    rs = np.random.RandomState(seed)
    while len(picks) < 64 or n_random > 0:
        i = int(rs.randint(n))
        if i not in picks:
            add(i, "random")
            n_random -= 1
    return picks


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, required=True, choices=[0, 1, 2, 3, 4, 5],
                    help="index into workloads.CONFIGS: 0-4 = BASELINE.json configs, 5 = the Ni-like workload (SURVEY.md 8(f)2)")
    ap.add_argument("--call", type=int, default=0, help="configs[1]: index of the call in the displacement sequence")
    ap.add_argument("--procs", type=int, default=os.cpu_count())
    ap.add_argument("--search", default="cells", choices=["cells", "brute"])
    ap.add_argument("--check-brute", type=int, default=16, help="random atoms whose row is re-checked by brute force")
    ap.add_argument("--random-atoms", type=int, default=24)
    ap.add_argument("--tmp", default="/tmp/nnp_golden")
    ap.add_argument("--out", default=None)
    args = ap.parse_args()

    t_start = time.time()
    cfg, sysm, model, pos = system_of(args.config, args.call)
    n = sysm.n_atoms
    tmp = os.path.join(args.tmp, "%s_call%d" % (cfg.name, args.call))
    os.makedirs(tmp, exist_ok=True)
    bounds = shard_bounds(n)
    tasks, results = mp.Queue(), mp.Queue()
    for s in range(N_SHARDS):
        if bounds[s + 1] > bounds[s]:
            tasks.put((s, bounds[s], bounds[s + 1]))
    procs = max(1, min(args.procs, N_SHARDS))
    for _ in range(procs):
        tasks.put(None)
    workers = [mp.Process(target=_worker, args=(w, args.config, args.call, args.search, tasks, results, tmp))
               for w in range(procs)]
    for p in workers:
        p.start()
    e_atom = np.zeros(n)
    cnt = np.zeros(n, dtype=np.int32)
    cnt0 = np.zeros(n, dtype=np.int32)
    sh_hash, sh_pairs = [0] * N_SHARDS, [0] * N_SHARDS
    t_nbr = t_rest = 0.0
    done_workers, done_shards = 0, 0
    while done_workers < procs:
        r = results.get()
        if r[0] == "done":
            done_workers += 1
            continue
        s, lo, hi, ea, c, c0, h, npairs, tn, tr = r
        e_atom[lo:hi] = ea; cnt[lo:hi] = c; cnt0[lo:hi] = c0
        sh_hash[s] = h; sh_pairs[s] = npairs
        t_nbr += tn; t_rest += tr
        done_shards += 1
        if done_shards % 16 == 0:
            print("  %d / %d shards, %.0f s" % (done_shards, N_SHARDS, time.time() - t_start), file=sys.stderr, flush=True)
    for p in workers:
        p.join()
    F = np.zeros((n, 3))
    for w in range(procs):
        f = os.path.join(tmp, "F_worker_%d.npy" % w)
        F += np.load(f)
        os.remove(f)
    wall_sweep = time.time() - t_start

    # stratified atoms: second run of exactly those centres with the BRUTE-FORCE scan (the definition)
    picks = stratify(pos, sysm.types, sysm.box, model.rc, cnt, cnt0, args.random_atoms, 1000 + args.config)
    atoms = np.array(sorted(picks), dtype=np.int64)
    om = oracle.OracleModel(model)
    rb = oracle.centres(om, pos, sysm.types, sysm.box, atoms, forces=False, want_g=True, search="brute", rows=True)
    assert np.array_equal(rb.e_atom, e_atom[atoms]), "cells and brute-force runs differ in E_i"
    assert np.array_equal(rb.nbr_count, cnt[atoms]), "cells and brute-force rows differ"
    rc_rows = oracle.neighbor_rows(pos, sysm.box, model.rc, atoms, "cells")
    for q in range(len(atoms)):
        assert np.array_equal(rc_rows[q], rb.row_idx[rb.row_off[q]:rb.row_off[q + 1]])
    extra = np.sort(np.random.RandomState(77 + args.config).choice(n, min(args.check_brute, n), replace=False))
    ra = oracle.neighbor_rows(pos, sysm.box, model.rc, extra, "brute")
    rc2 = oracle.neighbor_rows(pos, sysm.box, model.rc, extra, "cells")
    for x, y in zip(ra, rc2):
        assert np.array_equal(x, y)

    q_dig = [float(np.sum(F * digest_vectors(n, k))) for k in range(4)]
    out = {
        "about": "whole-system CPU-oracle results; written by tests/golden/make_fullsize_golden.py (imports oracle/ and "
                 "workloads/ only); see that file for the meaning of every field",
        "command": "python tests/golden/make_fullsize_golden.py " + " ".join(sys.argv[1:]),
        "config": cfg.name, "config_index": args.config, "call": args.call, "n_atoms": n, "model": model.name,
        "box": [float(x) for x in sysm.box], "rc": float(model.rc),
        "search": args.search,
        "rows_rechecked_by_brute_force": [int(i) for i in atoms] + [int(i) for i in extra],
        "cores": procs, "wall_s": round(time.time() - t_start, 1), "wall_s_sweep": round(wall_sweep, 1),
        "cpu_s_neighbour_search": round(t_nbr, 1), "cpu_s_sf_mlp_forces": round(t_rest, 1),
        "host_cpu": _cpu_name(),
        "e_total": math.fsum(e_atom),
        "e_abs_sum": math.fsum(np.abs(e_atom)),
        "e_atom_max_abs": float(np.abs(e_atom).max()),
        "n_pairs": int(np.sum(cnt, dtype=np.int64)),
        "nbr_hash": "%016x" % (sum(sh_hash) & ((1 << 64) - 1)),
        "nbr_count_hist": np.bincount(cnt).tolist(),
        "sum_f": [math.fsum(F[:, c]) for c in range(3)],
        "f_max_abs": float(np.abs(F).max()),
        "force_digest": {"seed": DIGEST_SEED, "values": q_dig,
                         "q_l1": [float(np.abs(digest_vectors(n, k)).sum()) for k in range(4)]},
        "shards": {
            "bounds": bounds,
            "e_sum": [math.fsum(e_atom[bounds[s]:bounds[s + 1]]) for s in range(N_SHARDS)],
            "f_sum": [[math.fsum(F[bounds[s]:bounds[s + 1], c]) for c in range(3)] for s in range(N_SHARDS)],
            "n_pairs": sh_pairs,
            "nbr_hash": ["%016x" % h for h in sh_hash],
        },
        "atoms": [{"index": int(m), "why": picks[int(m)],
                   "row": [int(j) for j in rb.row_idx[rb.row_off[q]:rb.row_off[q + 1]]],
                   "e_atom": float(rb.e_atom[q]),
                   "G": [float(x) for x in rb.G[q, :model.n_sf_per_elem[int(sysm.types[m])]]],
                   "F": [float(x) for x in F[m]]} for q, m in enumerate(atoms)],
    }
    name = "fullsize_%s%s.json" % (cfg.name, "_call%d" % args.call if args.call else "")
    path = args.out or os.path.join(HERE, name)
    with open(path, "w") as fh:
        json.dump(out, fh, indent=None, separators=(",", ":"))
        fh.write("\n")
    print("wrote %s: E_total = %.15g, %d atoms, %d stratified, %.0f s on %d processes"
          % (path, out["e_total"], n, len(atoms), time.time() - t_start, procs))


def _cpu_name():
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


if __name__ == "__main__":
    main()
