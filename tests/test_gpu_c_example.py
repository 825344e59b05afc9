"""The C ABI from plain C: examples/c_api_example.c is compiled with gcc against include/nnp.h and the in-tree
libnnp_b200.so, run on the GPU, and its printed energies and forces are compared with the CPU oracle on the same inputs
(the example's 64-bit LCG is restated here; no value is taken from the CUDA path)."""
import os
import subprocess

import numpy as np
import pytest

import oracle
import workloads as W
from workloads.model import SF_DTYPE, Model

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


class _Lcg:
    def __init__(self):
        self.s = 2002000054

    def uniform(self):
        self.s = (self.s * 6364136223846793005 + 1442695040888963407) % (1 << 64)
        return float(self.s >> 11) * (1.0 / 9007199254740992.0)


def _inputs():
    g = _Lcg()
    box = np.array([13.0, 14.5, 12.5])
    n = 240
    pos = np.zeros((n, 3))
    types = np.zeros(n, dtype=np.int32)
    for i in range(n):
        for c in range(3):
            pos[i, c] = g.uniform() * box[c]
        types[i] = 1 if i % 3 == 0 else 0
    rows = []
    for c in range(2):
        for e1 in range(2):
            rows.append((c, 2, e1, 0, 0.02, 0.0, 0.0, 0.0))
            rows.append((c, 2, e1, 0, 0.30, 1.0, 0.0, 0.0))
        rows.append((c, 3, 0, 0, 0.003, 0.0, 1.0, 1.0))
        rows.append((c, 3, 0, 1, 0.003, 0.0, -1.0, 2.0))
        rows.append((c, 3, 1, 1, 0.003, 0.0, 1.0, 4.0))
        rows.append((c, 3, 0, 1, 0.010, 0.0, 1.0, 2.0))
        rows.append((c, 9, 0, 0, 0.010, 0.0, -1.0, 1.0))
    nw = 6 * 9 + 6 + 6 + 1
    w0 = np.array([(g.uniform() - 0.5) * 0.6 for _ in range(nw)])
    w1 = np.array([(g.uniform() - 0.5) * 0.6 for _ in range(nw)])
    model = Model(elements=("H", "O"), rc=6.0, sf=np.array(rows, dtype=SF_DTYPE), layer_sizes=[[9, 6, 1], [9, 6, 1]],
                  weights=[w0, w1], name="c_example", n_sf_per_elem=[9, 9])
    return pos, types, box, model


def test_c_program_against_oracle(tmp_path):
    exe = str(tmp_path / "c_api_example")
    libdir = os.path.join(ROOT, "paper_2002_00054_b200")
    assert os.path.exists(os.path.join(libdir, "libnnp_b200.so")), "build the library first (__graft_entry__.build())"
    subprocess.run(["gcc", "-O2", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"),
                    os.path.join(ROOT, "examples", "c_api_example.c"), "-L", libdir, "-lnnp_b200",
                    "-Wl,-rpath," + libdir, "-lm", "-o", exe], check=True)
    r = subprocess.run([exe], capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr
    lines = r.stdout.strip().splitlines()
    head = lines[0].split()
    assert head[0] == "version" and head[2] == "kernels"
    assert (int(head[3]), int(head[4])) == (5, 5)           # NNP_KERNELS_MULTI: a narrow and a wide pass per element
    assert int(head[6]) > 10                                # kernels were launched
    e_total = float(lines[1].split()[1])
    rows = np.array([[float(x) for x in ln.split()[2:]] for ln in lines[2:242]])
    assert lines[242] == "repeat same"
    pos, types, box, model = _inputs()
    ref = oracle.compute(oracle.OracleModel(model), pos, types, box)
    assert abs(e_total - ref.e_total) <= 1e-10 * abs(ref.e_total)
    assert np.all(np.abs(rows[:, 0] - ref.e_atom) <= 1e-10 * np.abs(ref.e_atom).max())
    assert np.abs(rows[:, 1:] - ref.F).max() <= 1e-8
    assert np.abs(ref.F).max() > 1e-3
