"""Host logic of bench.py's roofline object (CPU only): the frozen denominators of roofline_counts.json are what
roofline_counts.py's operation lists give, and the ncu launch list committed under profiles/ is parsed into the
`traffic` / `fp64_pipe_pct` fields of the bench line."""
import json
import os

import pytest

import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_frozen_counts_match_the_operation_lists():
    import roofline_counts as rc
    frozen = json.load(open(os.path.join(ROOT, "roofline_counts.json")))
    for cfg in W.CONFIGS:
        _, model = W.build(W.Config(cfg.name, 4 if cfg.kind == "water" else 2, cfg.wide, 1, 1, cfg.seed_weights, None, cfg.kind))
        key = model.name if cfg.kind == "water" else "metal20"
        lists = rc.operation_lists(rc.table_shape(model))
        lists["network"] = rc.mlp_list(model.layer_sizes[0])
        units = {u: int(sum(c for _, c in ops)) for u, ops in lists.items()}
        assert units == frozen["models"][key]["unit_costs"]
        c = frozen["configs"][cfg.name]
        st, pa = c["statistics"], c["per_atom"]
        sf = st["neighbours"] * units["pair_forward"] + st["enumerated"] * units["enumerated_jk"] + st["contributing"] * units["triplet_forward"]
        fo = st["neighbours"] * units["pair_force"] + st["enumerated"] * units["enumerated_jk"] + st["contributing"] * units["triplet_force"]
        assert pa["sf"] == pytest.approx(sf, abs=0.06) and pa["force"] == pytest.approx(fo, abs=0.06)
        assert pa["total"] == pytest.approx(pa["sf"] + pa["mlp"] + pa["force"], abs=0.2)
    # the re-derived count of the headline config stays within SURVEY.md's +-15 % of its paper estimate
    tot = frozen["configs"]["large2M"]["per_atom"]["total"]
    assert abs(tot - 637e3) < 0.15 * 637e3
    # statistics come from the seeded system, not the ideal gas: close to, not equal to, 91 / 4,141 / 1,941
    st = frozen["configs"]["large2M"]["statistics"]
    assert 90 < st["neighbours"] < 92 and 4000 < st["enumerated"] < 4300 and 1850 < st["contributing"] < 2000


def test_ncu_launch_list_is_parsed_for_the_dominant_kernel():
    import bench
    m, src = bench._ncu_launch_metrics(3, r"k_force2<|k_force_small<")
    assert m is not None, src
    assert src.startswith("profiles/") and src.endswith("launches_config3.csv")
    assert 1e9 < m["dram_bytes"] < 1e10                      # a few GB per launch at 2.1 M atoms
    assert 50 < m["ncu_kernel_ms_cold"] < 120
    if m["fp64_pipe_pct"] is not None:
        assert 20 < m["fp64_pipe_pct"] < 100
        per_atom = m["fp64_warp_instr_executed"] * 32 / 2097153
        assert 2e5 < per_atom < 5e5                          # executed FP64 thread-instructions per atom (algorithmic: 396 k)
    assert bench._ncu_launch_metrics(0, "k_force2<")[0] is None           # no list committed for configs[0]: null with a reason
