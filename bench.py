"""bench.py -- NNP energy+force throughput on B200 (BASELINE.json metric: atom-steps/s + roofline fraction).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config k] [--impl ours|reference]

A "step" is one pass of the whole hot path (S0 sort .. S5 reduce, neighbour list rebuilt every
call) over one synthetic water-like system.  Default workload = BASELINE.json configs[3]
(2,097,153 atoms, base-52 model): the configuration the north-star target is quoted on; it fits
one GPU.  N > 1 (torchrun): the path does not shard in this build ("replicas only", DESIGN.md
section 8(e)) -> every rank evaluates the same system on its own GPU, value = N * atoms * K / max time.

One JSON line on stdout (rank 0).  Extra keys: roofline (dominant kernel k_force2, FP64-ALU bound; `frac` on the
frozen count of roofline_counts.json, `frac_survey_estimate` on SURVEY.md's paper estimate, `fp64_pipe_pct` /
`traffic` parsed from the newest committed ncu launch list), cpu_baseline (the oracle on a bounded sample of
centres of the same system), e2e (host buffers through nnp_compute_host), clocks, gpu_launches, stage_ms,
config_sweep (short timed runs of configs[1], [2], [4]).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "nnp_energy_force_atom_steps_per_sec"
UNIT = "atom-steps/s"

# Algorithmic FP64-pipe thread-instructions per atom-step: roofline_counts.json, written by roofline_counts.py
# (operation lists of the minimal per-centre evaluation scheme x statistics measured on the seeded systems;
# DESIGN.md "Roofline denominators").  SURVEY.md 8(d)'s paper estimate (+-15 %) is reported beside it.
def _roofline_counts():
    with open(os.path.join(ROOT, "roofline_counts.json")) as fh:
        return json.load(fh)


def _ncu_launch_metrics(cfg_index: int, kernel: str):
    """Per-launch ncu metrics of `kernel` from the newest committed launch list of this config
    (profiles/*launches_config<k>.csv, written by the ncu command its .md names): DRAM bytes and, when the
    list carries them, FP64-pipe utilisation and executed FP64 warp-instructions.  -> (dict, source) or (None, why)."""
    import csv
    import glob
    files = sorted(glob.glob(os.path.join(ROOT, "profiles", "*launches_config%d.csv" % cfg_index)))
    if not files:
        return None, "no profiles/*launches_config%d.csv committed" % cfg_index
    path = files[-1]
    per = {}
    with open(path, newline="") as fh:
        rows = [r for r in csv.reader(l for l in fh if l.startswith('"'))]
    if not rows:
        return None, "no rows in " + os.path.basename(path)
    head = rows[0]
    try:
        ik, im, iv, iid = head.index("Kernel Name"), head.index("Metric Name"), head.index("Metric Value"), head.index("ID")
    except ValueError:
        return None, "unexpected header in " + os.path.basename(path)
    import re
    pat = re.compile(kernel)
    for r in rows[1:]:
        if len(r) <= iv or not pat.search(r[ik]):
            continue
        try:
            per.setdefault(r[im], {})[r[iid]] = float(r[iv].replace(",", ""))
        except ValueError:
            pass
    if "dram__bytes_read.sum" not in per:
        return None, "no %s launch with DRAM metrics in %s" % (kernel, os.path.basename(path))
    mean = {k: sum(v.values()) / len(v) for k, v in per.items()}
    out = {"dram_bytes": mean["dram__bytes_read.sum"] + mean.get("dram__bytes_write.sum", 0.0),
           "launches_averaged": len(per["dram__bytes_read.sum"]),
           "ncu_kernel_ms_cold": mean.get("gpu__time_duration.sum", float("nan")) / 1e6}
    k = "sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_active"
    out["fp64_pipe_pct"] = mean.get(k)
    k = "sm__inst_executed_pipe_fp64.sum"
    out["fp64_warp_instr_executed"] = mean.get(k)
    return out, "profiles/" + os.path.basename(path)


# FP64 pipe peak derived from unit counts and clocks: 148 SMs x 64 DFMA lanes/clk x clocks.max.sm
FP64_LANES_PER_SM = 64
N_SM = 148


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        return json.load(open(p))
    except Exception:
        return {}


def max_over_ranks(x: float, device=None) -> float:
    """MAX of a per-rank scalar over the process group (identity when not initialised)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(x)
    t = torch.tensor([float(x)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_value(n_atoms: int, steps: int, world: int, ms_max: float) -> float:
    """Whole-job atom-steps/s of `world` independent replicas ("replicas only"):
    every rank evaluates n_atoms atoms `steps` times; the job ends when the slowest rank ends."""
    return world * n_atoms * steps / (ms_max * 1e-3)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.rows = []
        self.proc = None
        self.thread = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                 "-lms", "200"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        def pump():
            for line in self.proc.stdout:
                self.rows.append(line.strip())
        self.thread = threading.Thread(target=pump, daemon=True)
        self.thread.start()

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, smax, power, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for r in self.rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); smax.append(float(f[1])); power.append(float(f[2]))
            except ValueError:
                continue
            for k, nm in enumerate(names):
                if f[3 + k].lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(smax)), "power_w_max": float(max(power)),
                "samples": len(sm), "reasons": sorted(reasons)}


def oracle_sample(cfg_index: int, n_centres: int, seed: int = 12345):
    """Time the CPU oracle, as it stands, on `n_centres` randomly chosen centres of the workload:
    brute-force neighbour search + SFs + network + force contributions of each centre
    (= n_centres atom-steps).  -> (seconds, seconds in the neighbour search, cores)."""
    import oracle
    import workloads as W
    sysm, model = W.build(W.CONFIGS[cfg_index])
    om = oracle.OracleModel(model)
    rs = np.random.RandomState(seed)
    sel = np.sort(rs.choice(sysm.n_atoms, min(n_centres, sysm.n_atoms), replace=False)).astype(np.int64)
    t0 = time.perf_counter()
    r = oracle.centres(om, sysm.pos, sysm.types, sysm.box, sel, forces=True, want_g=False)
    dt = time.perf_counter() - t0
    return dt, float(r.timing[0]), 1, int(sel.size)


def sweep_config(k: int, local: int, peak_alu: float, counts: dict, steps: int = 5, warmup: int = 3):
    """Short timed run (CUDA events on the launching stream, device-resident inputs, `warmup` untimed + `steps`
    timed evaluations) of another BASELINE.json config, so that the driver's record carries every config."""
    import torch

    import workloads as W
    from paper_2002_00054_b200 import NNP
    cfg = W.CONFIGS[k]
    sysm, model = W.build(cfg)
    n = sysm.n_atoms
    dev = torch.device("cuda", local)
    nnp = NNP.from_model(model, device=local)
    pos = torch.tensor(sysm.pos, dtype=torch.float64, device=dev)
    typ = torch.tensor(sysm.types, dtype=torch.int32, device=dev)
    out = (torch.empty(n, dtype=torch.float64, device=dev), torch.empty(1, dtype=torch.float64, device=dev),
           torch.empty((n, 3), dtype=torch.float64, device=dev))
    disp = None
    if cfg.seed_disp is not None:
        disp = [torch.tensor(W.displacement(n, cfg.seed_disp, c + 1), device=dev) for c in range(4)]

    def step(i):
        if disp is not None:
            pos.add_(disp[i % len(disp)])
        nnp.compute(pos, typ, sysm.box, out=out, sync=False)

    for i in range(warmup):
        step(i)
    nnp.sync_status()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for i in range(steps):
        step(i)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / steps
    nnp.sync_status()
    nnp.set_timing(True)
    stage = np.zeros(6)
    for i in range(steps):
        step(i)
        tm = nnp.timings_ms()
        stage += np.array([tm[q] for q in ("sort", "neighbors", "symmetry_functions", "networks", "forces", "finalize")])
    stage /= steps
    nnp.set_timing(False)
    ws = nnp.workspace_bytes(n)
    nnp.close()
    instr = counts["configs"][cfg.name]["per_atom"]
    return {"config_index": k, "workload": cfg.name, "n_atoms": n, "model": model.name, "steps": steps, "warmup": warmup,
            "value": n / (ms * 1e-3), "unit": UNIT, "ms_per_step": ms,
            "stage_ms": {"neighbors": float(stage[1]), "symmetry_functions": float(stage[2]), "networks": float(stage[3]),
                         "forces": float(stage[4])},
            "roofline_frac_whole_step": instr["total"] * n / (ms * 1e-3) / peak_alu,
            "roofline_frac_k_force2": instr["force"] * n / (float(stage[4]) * 1e-3) / peak_alu,
            "l2": "workspace %.0f MB %s the 126 MB L2" % (ws / 1e6, "exceeds" if ws > 126e6 else "fits in")}


def n2p2like_model():
    """Probe table of `--table n2p2like` (the one tests/test_gpu_parity.py::test_multi_pass_tables checks)."""
    import workloads as W
    from workloads.model import Model, mlp_weights
    rows, rcs = [], []
    for c in range(2):
        for e1 in range(2):
            for (eta, rs, rr) in ((0.003, 0.0, 6.0), (0.03, 0.0, 6.0), (0.2, 1.0, 4.5), (0.6, 2.0, 3.5)):
                rows.append((c, 2, e1, 0, eta, rs, 0.0, 0.0)); rcs.append(rr)
        for (e1, e2) in ((0, 0), (0, 1), (1, 1)):
            for ie, eta in enumerate((0.0005, 0.002, 0.004, 0.008, 0.015, 0.03, 0.07)):
                for lam in (1.0, -1.0):
                    for zeta in (1.0, 4.0):
                        rows.append((c, 3, e1, e2, eta, 0.0, lam, zeta)); rcs.append(6.0 if ie < 5 else 4.8)
    sf = np.array(rows, dtype=W.SF_DTYPE)
    n_per = [int(np.sum(sf["central"] == c)) for c in range(2)]
    layer_sizes = [[n_per[c], 25, 25, 1] for c in range(2)]
    return Model(elements=("H", "O"), rc=6.0, sf=sf, layer_sizes=layer_sizes,
                 weights=[mlp_weights(layer_sizes[c], 200200154, c) for c in range(2)], name="n2p2like92",
                 n_sf_per_elem=n_per, sf_cutoffs=rcs)


def run_reference(args):
    """--impl reference: the oracle on the host cores, each step a bounded sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import oracle
    import workloads as W
    cfg = W.CONFIGS[args.config]
    sysm, model = W.build(cfg)
    om = oracle.OracleModel(model)
    # ~50 ms per centre at 2.1 M atoms (O(N) neighbour scan each): keep the whole run to a few minutes
    per_step = args.ref_centres
    if per_step <= 0:
        budget_s = 120.0
        est = 2.5e-8 * sysm.n_atoms + 1.2e-2
        per_step = int(max(4, min(512, budget_s / ((args.steps + args.warmup) * est))))
    rs = np.random.RandomState(777)

    def step():
        sel = np.sort(rs.choice(sysm.n_atoms, min(per_step, sysm.n_atoms), replace=False)).astype(np.int64)
        oracle.centres(om, sysm.pos, sysm.types, sysm.box, sel, forces=True, want_g=False)
        return sel.size

    for _ in range(args.warmup):
        step()
    t0 = time.perf_counter()
    done = 0
    for _ in range(args.steps):
        done += step()
    dt = time.perf_counter() - t0
    value = done / dt
    sample = "%d randomly chosen centres of %s per step (brute-force neighbours + SF + MLP + forces each)" % (
        per_step, cfg.name)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        # the same keys as the CUDA arm's config (workload, atoms and model are the same; the rest describes this arm)
        "config": {"workload": cfg.name, "n_atoms": sysm.n_atoms, "model": model.name, "kernels": ["oracle"] * len(model.elements),
                   "box": float(sysm.box[0]), "neighbor_rebuild": "every call (brute-force scan per centre)", "md": False,
                   "parallelism": "1 host core (single-threaded oracle)", "l2": "n/a (host)"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3, help="index into BASELINE.json configs (default 3 = 2.1 M atoms)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--ref-centres", type=int, default=0, help="--impl reference: centres per step (0 = auto)")
    ap.add_argument("--cpu-centres", type=int, default=400, help="oracle sample size of the cpu_baseline leg (0 = skip)")
    ap.add_argument("--md", action="store_true",
                    help="time velocity-Verlet MD steps (nnp_md_run: kick+drift, the whole path, kick) instead of bare evaluations")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--table", default="baseline", choices=["baseline", "free", "generic", "zeta5", "queue", "n2p2like", "wide9"],
                    help="SF table probe (not a BASELINE.json workload): 'free' breaks the eta ratio of the angular set "
                         "(0.01 -> 0.0123: lane-owned kernels with per-eta exponentials), 'generic' also replaces zeta 16 by 3 "
                         "(round 1: queue-based generic kernels; now one pass with the exponent menu 1, 2, 4; 3), 'zeta5' replaces "
                         "zeta 4 by 5 as well (two passes), 'queue' also lists one angular function twice, which no "
                         "pass menu holds (the queue-based generic kernels), 'n2p2like' is a table shaped like published n2p2 models (zeta in {1, 4}, "
                         "seven eta values, lambda = +-1, angular functions of two cutoff radii: 3 passes of the free-eta "
                         "kernels), 'wide9' turns the angular functions of the smaller eta into wide ones (n2p2 kind 9: one narrow and one "
                         "wide pass); the roofline object is then not meaningful")
    ap.add_argument("--skin", type=float, default=0.0,
                    help="probe of what a Verlet-skin neighbour list would cost the hot kernels: the neighbour list is built "
                         "with rc + SKIN while every symmetry function keeps its cutoff (nnp_set_sf_cutoffs), i.e. exactly the "
                         "list a skin scheme would hand the kernels on its reuse steps; the list is still rebuilt every call")
    ap.add_argument("--reuse-skin", type=float, default=0.0,
                    help="nnp_set_neighbor_skin: keep a candidate list of radius rc + SKIN across calls and filter the exact list "
                         "from it; rebuilt when an atom has moved SKIN/2 (decided on the device).  Not the headline: BASELINE.json's "
                         "metric rebuilds the list every call.  With static positions (no --md) no timed call rebuilds")
    ap.add_argument("--max-neighbors", type=int, default=0, help="nnp_set_max_neighbors (0: the default; the Ni-like config 5 uses 24)")
    ap.add_argument("--deterministic", action="store_true",
                    help="nnp_set_deterministic_forces: fixed-point force accumulation (bit-reproducible forces)")
    ap.add_argument("--no-probe", action="store_true", help="skip the DFMA issue-rate probe (for ncu runs)")
    ap.add_argument("--no-sweep", action="store_true",
                    help="skip the short timed runs of configs[1], [2], [4] that the default line carries as config_sweep")
    ap.add_argument("--precision", default="f64", choices=["f64", "mixed"],
                    help="arithmetic mode of the hot kernels: f64 (headline) or the opt-in mixed mode of nnp_set_precision "
                         "(FP32 staging and per-triplet arithmetic, FP64 accumulation; not a BASELINE.json result)")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist

    import workloads as W
    from paper_2002_00054_b200 import NNP, measure_fp64_peak
    from paper_2002_00054_b200.binding import table_kernels

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    cfg = W.CONFIGS[args.config]
    sysm, model = W.build(cfg)
    if args.table == "n2p2like":
        model = n2p2like_model()
    elif args.table == "wide9":
        ang = model.sf["kind"] == 3
        model.sf["kind"][ang & (model.sf["eta"] == model.sf["eta"][ang].min())] = 9
        model.name += "+wide9"
    elif args.table != "baseline":
        ang = model.sf["kind"] == 3
        model.sf["eta"][ang & (model.sf["eta"] == 0.01)] = 0.0123
        if args.table in ("generic", "zeta5", "queue"):
            model.sf["zeta"][ang & (model.sf["zeta"] == 16.0)] = 3.0
        if args.table == "zeta5":
            model.sf["zeta"][ang & (model.sf["zeta"] == 4.0)] = 5.0
        if args.table == "queue":
            for c in range(len(model.elements)):
                q = np.nonzero(ang & (model.sf["central"] == c))[0]
                for key in ("eta", "lam", "zeta", "e1", "e2"):
                    model.sf[key][q[1]] = model.sf[key][q[0]]
        model.name += "+" + args.table
    if args.skin > 0.0:
        rc_sf = list(model.sf_cutoffs) if model.sf_cutoffs is not None else [model.rc] * len(model.sf)
        model.rc = model.rc + args.skin
        model.sf_cutoffs = rc_sf
        model.name += "+skin%g" % args.skin
    n = sysm.n_atoms
    nnp = NNP.from_model(model, device=local)
    if args.precision != "f64":
        nnp.set_precision(args.precision)
    if args.deterministic:
        nnp.set_deterministic_forces(True)
    if cfg.kind == "metal":
        nnp.set_max_neighbors(args.max_neighbors or 24)      # 18 neighbours per atom: the 8-lanes-per-centre kernels of k_small.cu (24 slots)
    if args.reuse_skin > 0.0:
        nnp.set_neighbor_skin(args.reuse_skin)
    pos = torch.tensor(sysm.pos, dtype=torch.float64, device=dev)
    typ = torch.tensor(sysm.types, dtype=torch.int32, device=dev)
    out = (torch.empty(n, dtype=torch.float64, device=dev), torch.empty(1, dtype=torch.float64, device=dev),
           torch.empty((n, 3), dtype=torch.float64, device=dev))
    # configs[1]: small random displacements between calls (cumulative, applied on the device copy)
    disp = None
    if cfg.seed_disp is not None:
        disp = [torch.tensor(W.displacement(n, cfg.seed_disp, c + 1), device=dev) for c in range(4)]

    vel = None
    if args.md:     # thermal-ish velocities (sigma 0.005 A/fs), masses of H and O; forces of the start positions
        g = torch.Generator(device=dev).manual_seed(1234)
        vel = 0.005 * torch.randn((n, 3), dtype=torch.float64, device=dev, generator=g)
        nnp.compute(pos, typ, sysm.box, out=out, sync=True)

    def step(i):
        if args.md:
            nnp.md_run(1, 0.25, (1.008, 15.999), pos, vel, typ, sysm.box, out, sync=False)
            return
        if disp is not None:
            pos.add_(disp[i % len(disp)])
        nnp.compute(pos, typ, sysm.box, out=out, sync=False)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # FP64 issue-rate probe (roofline context), before the timed region
    dfma_burst, dfma_sust = (float("nan"), float("nan")) if args.no_probe else measure_fp64_peak(local, 0.5)

    for i in range(args.warmup):
        step(i)
    nnp.sync_status()
    nnp.set_timing(True)
    stage_ms = np.zeros(6)
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    barrier()
    e0 = torch.cuda.Event(enable_timing=True)
    e1 = torch.cuda.Event(enable_timing=True)
    launches = 0
    e0.record()
    for i in range(args.steps):
        step(i)
        launches += nnp.last_launch_count()
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    # stage times of the LAST timed step (events recorded on the stream inside nnp_compute)
    t_last = nnp.timings_ms()
    clocks = sampler.stop() if rank == 0 else None
    nnp.sync_status()
    nnp.set_timing(False)
    ms = max_over_ranks(ms, dev)
    rebuild_note = "every call"
    if args.reuse_skin > 0.0:
        calls, rebuilds = nnp.neighbor_rebuilds()
        rebuild_note = "skin %.2f A: %d rebuilds in %d calls (warm-up included)" % (args.reuse_skin, rebuilds, calls)

    # per-stage average over K more (untimed for the headline) steps, events inside nnp_compute
    nnp.set_timing(True)
    for i in range(args.steps):
        step(i)
        tm = nnp.timings_ms()
        stage_ms += np.array([tm[k] for k in ("sort", "neighbors", "symmetry_functions", "networks", "forces", "finalize")])
    stage_ms /= args.steps
    nnp.set_timing(False)

    # end to end: HOST buffers through nnp_compute_host (h2d + compute + d2h inside the call)
    e2e = None
    if not args.no_e2e:
        hp = torch.tensor(sysm.pos, dtype=torch.float64).pin_memory()
        ht = torch.tensor(sysm.types, dtype=torch.int32).pin_memory()
        he = torch.empty(n, dtype=torch.float64).pin_memory()
        hE = torch.empty(1, dtype=torch.float64).pin_memory()
        hf = torch.empty((n, 3), dtype=torch.float64).pin_memory()
        for _ in range(2):
            nnp.compute_host(hp, ht, sysm.box, out=(he, hE, hf))
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            nnp.compute_host(hp, ht, sysm.box, out=(he, hE, hf))
        dt = time.perf_counter() - t0
        dt = max_over_ranks(dt, dev)
        e2e = {"value": job_value(n, args.steps, world, dt * 1e3), "unit": UNIT, "h2d_bytes_per_step": n * 28,
               "d2h_bytes_per_step": n * 32 + 8, "ms_per_step": 1e3 * dt / args.steps,
               "api": "nnp_compute_host (pinned host buffers)"}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    peaks = _peaks()
    sm_max = float(peaks.get("sm_max_mhz", 1965.0))
    peak_alu = N_SM * FP64_LANES_PER_SM * sm_max * 1e6
    counts = _roofline_counts()
    instr = counts["configs"][cfg.name]["per_atom"]
    survey = counts["survey_estimate_per_atom"].get(counts["configs"][cfg.name]["model"])
    force_ms = float(stage_ms[4])
    step_s = ms / args.steps * 1e-3
    achieved = instr["force"] * n / (force_ms * 1e-3)
    total_instr = instr["total"] * n
    hbm_bytes_per_atom = 1.0e3 if cfg.kind == "metal" else (2.8e3 if not cfg.wide else 5.2e3)
    # the dominant kernel: k_force2<...> (not its list-driven sibling for the few big centres), k_force_small on the metal workload
    baseline_table = args.table == "baseline" and args.precision == "f64" and args.skin == 0.0 and args.reuse_skin == 0.0
    if baseline_table:
        ncu, ncu_src = _ncu_launch_metrics(args.config, r"k_force2<|k_force_small<")
    else:
        ncu, ncu_src = None, "the committed launch lists are of the FP64 run on BASELINE.json's tables"
    roofline = {
        "bound": "alu", "kernel": "k_force_small" if cfg.kind == "metal" else "k_force2", "achieved": achieved / 1e12, "peak": peak_alu / 1e12,
        "unit": "T FP64 instr/s", "frac": achieved / peak_alu,
        "frac_is": "algorithmic-model fraction: frozen FP64 instruction count of the minimal per-centre scheme "
                   "(roofline_counts.json) / kernel time / derived pipe peak; the hardware pipe utilisation is fp64_pipe_pct",
        "frac_survey_estimate": (survey["force"] * n / (force_ms * 1e-3) / peak_alu) if survey else None,
        "traffic": ncu["dram_bytes"] if ncu else None,
        "traffic_source": ncu_src,
        "traffic_algorithmic": (n * (8 * nnp.g_stride + 4 * 91 + 28 + 24)) if cfg.kind != "metal" else None,
        "fp64_pipe_pct": ncu["fp64_pipe_pct"] if ncu else None,
        "fp64_thread_instr_executed_per_atom": (ncu["fp64_warp_instr_executed"] * 32 / n
                                                if ncu and ncu["fp64_warp_instr_executed"] else None),
        "peak_source": "derived: 148 SMs x 64 FP64 lanes x %.0f MHz (clocks.max.sm); DFMA probe in this run: "
                       "burst %.2f, sustained %.2f T instr/s" % (sm_max, dfma_burst / 1e12, dfma_sust / 1e12),
        "frac_of_measured_dfma": achieved / dfma_burst,
        "algorithmic_instr_per_launch": instr["force"] * n,
        "kernel_ms": force_ms,
        "stages": {"sf": {"instr_per_atom": instr["sf"], "ms": float(stage_ms[2]),
                          "frac": instr["sf"] * n / (float(stage_ms[2]) * 1e-3) / peak_alu},
                   "mlp": {"instr_per_atom": instr["mlp"], "ms": float(stage_ms[3]),
                           "frac": instr["mlp"] * n / (float(stage_ms[3]) * 1e-3) / peak_alu},
                   "force": {"instr_per_atom": instr["force"], "ms": force_ms, "frac": achieved / peak_alu}},
        "whole_step": {"fp64_instr": total_instr, "frac": total_instr / step_s / peak_alu,
                       "frac_survey_estimate": (sum(survey.values()) * n / step_s / peak_alu) if survey else None,
                       "hbm_bytes": hbm_bytes_per_atom * n,
                       "hbm_frac": hbm_bytes_per_atom * n / step_s / (peaks.get("hbm_gbs", 6650.0) * 1e9)},
    }
    if not baseline_table:
        roofline["note"] = "probe table / precision mode: the frozen count is the base table's, fractions are indicative only"

    sweep = None
    if world == 1 and args.config == 3 and baseline_table and not args.md and not args.no_sweep:
        sweep = [sweep_config(k, local, peak_alu, counts) for k in (1, 2, 4)]

    cpu = None
    if args.cpu_centres > 0:
        dt, t_nbr, cores, ns = oracle_sample(args.config, args.cpu_centres)
        cpu = {"value": ns / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
               "value_without_neighbour_scan": ns / max(dt - t_nbr, 1e-9),
               "sample": "%d randomly chosen centres of %s, each: O(N) brute-force neighbour scan + SFs + MLP + "
                         "force contributions; %.1f s total, %.1f s of it in the O(N^2)-style neighbour scan no production "
                         "CPU code would use (value_without_neighbour_scan leaves it out)" % (ns, cfg.name, dt, t_nbr)}

    line = {
        "metric": METRIC, "value": job_value(n, args.steps, world, ms), "unit": UNIT, "n_gpus": world,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64" if args.precision == "f64" else "f32-stage/f64-acc", "data": "synthetic",
        "config": {"workload": cfg.name, "n_atoms": n, "model": model.name, "kernels": list(table_kernels(model)), "box": float(sysm.box[0]),
                   "neighbor_rebuild": rebuild_note, "md": bool(args.md),
                   "force_accumulation": "fixed-point 2^-40 eV/A (bit-reproducible)" if args.deterministic else "FP64 atomics", "parallelism": "replicas x%d" % world,
                   "l2": ("working set per step (%.2f GB workspace) %s the 126 MB L2; no flush between steps"
                          % (nnp.workspace_bytes(n) / 1e9, "exceeds" if nnp.workspace_bytes(n) > 126e6 else "FITS IN"))},
        "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "clocks": clocks, "gpu_launches": launches,
        "stage_ms": dict(zip(("sort", "neighbors", "symmetry_functions", "networks", "forces", "finalize"),
                             [float(x) for x in stage_ms])),
        "stage_ms_last_timed_step": t_last,
        "config_sweep": sweep,
    }
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
