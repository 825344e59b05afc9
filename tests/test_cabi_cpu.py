"""CPU-side checks of the C-ABI library: it loads, exports every symbol include/nnp.h declares,
and rejects bad arguments synchronously (no compute calls -- there is no GPU here)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    import __graft_entry__ as g
    from paper_2002_00054_b200 import build as b
    if not os.path.exists(b.LIB):
        g.build()
    from paper_2002_00054_b200 import load_library
    return load_library()


def test_exports_match_header(lib):
    from paper_2002_00054_b200 import EXPORTS
    hdr = open(os.path.join(ROOT, "include", "nnp.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(nnp_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(EXPORTS)
    for name in declared:
        assert getattr(lib, name) is not None
    assert lib.nnp_version().decode() == "0.1"


def _create(lib, model, n_elem=None, rc=None, sf=None, layer_sizes=None, weights=None):
    from paper_2002_00054_b200.binding import _SF
    n_elem = len(model.elements) if n_elem is None else n_elem
    sf = np.ascontiguousarray(model.sf if sf is None else sf)
    assert sf.dtype.itemsize == C.sizeof(_SF)
    layer_sizes = model.layer_sizes if layer_sizes is None else layer_sizes
    weights = model.weights if weights is None else weights
    names = (C.c_char_p * len(model.elements))(*[e.encode() for e in model.elements])
    nl = np.array([len(ls) - 1 for ls in layer_sizes], dtype=np.int32)
    lsa = [np.ascontiguousarray(ls, dtype=np.int32) for ls in layer_sizes]
    wa = [np.ascontiguousarray(w, dtype=np.float64) for w in weights]
    lsp = (C.c_void_p * len(lsa))(*[a.ctypes.data for a in lsa])
    wp = (C.c_void_p * len(wa))(*[a.ctypes.data for a in wa])
    h = C.c_void_p(None)
    st = lib.nnp_create(C.byref(h), n_elem, names, float(model.rc if rc is None else rc), int(sf.shape[0]),
                        sf.ctypes.data_as(C.c_void_p), nl.ctypes.data_as(C.c_void_p), lsp, wp, 0)
    return st, h


def test_create_rejects_bad_arguments(lib):
    model = W.make_model(False)
    INVALID = 1
    assert _create(lib, model, n_elem=0)[0] == INVALID
    assert _create(lib, model, n_elem=5)[0] == 8          # NNP_ERR_LIMIT: a compile-time limit, with its own message
    assert b"NNP_MAX_ELEMENTS" in lib.nnp_last_error(None)
    ls = [list(x) for x in model.layer_sizes]; ls[0][1] = 300
    w = [np.zeros(52 * 300 + 300 + 300 * 25 + 25 + 25 + 1), model.weights[1]]
    assert _create(lib, model, layer_sizes=ls, weights=w)[0] == 8
    assert b"256" in lib.nnp_last_error(None)
    assert _create(lib, model, rc=-1.0)[0] == INVALID
    sf = model.sf.copy(); sf["kind"][3] = 7
    assert _create(lib, model, sf=sf)[0] == INVALID
    sf = model.sf.copy(); sf["zeta"][20] = 2.5           # non-integer zeta
    assert _create(lib, model, sf=sf)[0] == INVALID
    assert b"zeta" in lib.nnp_last_error(None)
    sf = model.sf.copy(); sf["lam"][20] = 0.5
    assert _create(lib, model, sf=sf)[0] == INVALID
    sf = model.sf.copy(); sf["e1"][0] = 2
    assert _create(lib, model, sf=sf)[0] == INVALID
    sf = model.sf.copy(); sf["central"][0] = -1
    assert _create(lib, model, sf=sf)[0] == INVALID
    ls = [list(x) for x in model.layer_sizes]; ls[0][0] = 51
    assert _create(lib, model, layer_sizes=ls)[0] == INVALID
    ls = [list(x) for x in model.layer_sizes]; ls[1][-1] = 2
    assert _create(lib, model, layer_sizes=ls)[0] == INVALID


def test_kernel_choice_per_table(lib):
    """Host logic of nnp_create: which kernels a symmetry-function table runs on (no GPU involved)."""
    from conftest import tiny_model
    from paper_2002_00054_b200.binding import table_kernels, NNPError
    assert table_kernels(W.make_model(False)) == ("base12", "base12")
    assert table_kernels(W.make_model(True)) == ("wide32", "wide32")
    assert table_kernels(W.make_model(False, elements=("A", "B", "C"))) == ("base12",) * 3
    m = W.make_model(False)
    ang = m.sf["kind"] == 3
    m.sf["eta"][ang & (m.sf["eta"] == 0.01)] = 0.0123             # eta ratio broken: the free-eta menu kernels
    assert table_kernels(m) == ("free16", "free16")                 # two eta values: the 16-accumulator instantiation
    m3 = W.make_model(True)
    m3.sf["eta"][(m3.sf["kind"] == 3) & (m3.sf["eta"] == 0.003)] = 0.0041
    assert table_kernels(m3) == ("free32", "free32")               # four unrelated eta values
    m.sf["zeta"][ang & (m.sf["zeta"] == 16.0) & (m.sf["central"] == 1)] = 3.0     # zeta {1,2,4,3}: still ONE menu (zeta0 = 1, zeta_x = 3), one pass
    assert table_kernels(m) == ("free16", "free16")
    m.sf["zeta"][ang & (m.sf["zeta"] == 4.0) & (m.sf["central"] == 1)] = 5.0      # {1,2,5,3}: menus (1; 3) and (5): two passes, that element only
    assert table_kernels(m) == ("free16", "multi")
    m = W.make_model(False)
    m.sf["kind"][np.nonzero(ang)[0][0]] = 9                         # one wide angular SF on element 0: a pass of its own
    assert table_kernels(m) == ("multi", "base12")
    m.sf["zeta"][np.nonzero(ang)[0][0]] = 3.0                       # ... with zeta = 3: still a pass of its own (menu zeta0 = 3)
    assert table_kernels(m) == ("multi", "base12")
    m = W.make_model(False)
    q = np.nonzero(ang)[0][:5]
    m.sf["eta"][q] = [0.002, 0.003, 0.004, 0.005, 0.006]           # more than four eta values: several passes of the free-eta kernels
    assert table_kernels(m)[0] == "multi"
    rows = [(0, 2, 0, 0, 0.1, 0.0, 0.0, 0.0)] + [(0, 3, 0, 0, 0.01, 0.0, 1.0, float(z)) for z in (1, 2, 3, 4, 6, 8, 12, 16, 48, 64)]
    assert table_kernels(tiny_model(rows)) == ("multi",)            # menus (1,2,4;16), (3,6,12;48), (8;64): three passes
    rows = [(0, 2, 0, 0, 0.1, 0.0, 0.0, 0.0)] + [(0, 3, 0, 0, 0.01, 0.0, 1.0, float(z)) for z in (3, 5, 7, 9, 11, 13, 15, 17, 19)]
    assert table_kernels(tiny_model(rows)) == ("multi",)            # nine odd exponents: five menus of (zeta0; zeta_x)
    rows = [(0, 2, 0, 0, 0.1, 0.0, 0.0, 0.0)] + [(0, 3, 0, 0, 0.01, 0.0, 1.0, float(z)) for z in range(3, 64, 2)]
    assert table_kernels(tiny_model(rows)) == ("generic",)          # 31 odd exponents: 16 menus, more than 8 passes
    rows = [(0, 2, 0, 0, 0.1, 0.0, 0.0, 0.0)] + [(0, 3, 0, 0, 0.001 * (k + 1), 0.0, 1.0, 1.0) for k in range(33)]
    assert table_kernels(tiny_model(rows)) == ("generic",)          # 33 eta values: more than 8 passes of four
    m = W.make_model(False)
    q = np.nonzero(ang)[0]
    m.sf["zeta"][q[1]] = m.sf["zeta"][q[0]]; m.sf["lam"][q[1]] = m.sf["lam"][q[0]]; m.sf["eta"][q[1]] = m.sf["eta"][q[0]]
    assert table_kernels(m)[0] == "generic"                         # the same (eta, lambda, zeta) twice in one pair group
    rows = [(0, 2, 0, 0, 0.1, 0.0, 0.0, 0.0), (0, 3, 0, 0, 0.5, 0.0, 1.0, 2.0)]
    assert table_kernels(tiny_model(rows, rc=6.0)) == ("free16",)
    assert table_kernels(tiny_model(rows, rc=25.0)) == ("generic",)  # eta 3 rc^2 > 700: exp_small's range
    assert table_kernels(tiny_model(rows[:1])) == ("generic",)      # radial only
    bad = W.make_model(False)
    bad.sf["lam"][np.nonzero(ang)[0][0]] = 0.5
    with pytest.raises(NNPError):
        table_kernels(bad)


def test_create_without_gpu_reports_cuda_error(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    st, h = _create(lib, W.make_model(False))
    assert st == 6 and not h.value          # NNP_ERR_CUDA: no CPU fallback
    assert len(lib.nnp_last_error(None)) > 0


def test_null_model_calls_are_safe(lib):
    assert lib.nnp_workspace_bytes(None, 100) == 0
    assert lib.nnp_sync_status(None) == 1
    assert lib.nnp_g_stride(None) == 0
    lib.nnp_destroy(None)


def test_binding_fails_loudly_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2002_00054_b200 import NNP, NNPError
    with pytest.raises(NNPError):
        NNP.from_model(W.make_model(False))
