"""ctypes front end of the CPU oracle (oracle/nnp_oracle.c).

TEST INFRASTRUCTURE: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs import this.  It never imports the CUDA
package, and the CUDA package never imports it.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from .build import build as _build

_lib = None


class _SF(C.Structure):
    _fields_ = [("central", C.c_int32), ("kind", C.c_int32), ("e1", C.c_int32), ("e2", C.c_int32),
                ("eta", C.c_double), ("rs", C.c_double), ("lam", C.c_double), ("zeta", C.c_double)]


class _Model(C.Structure):
    _fields_ = [("n_elem", C.c_int32), ("rc", C.c_double), ("n_sf", C.c_int32),
                ("sf", C.c_void_p), ("n_layers", C.c_void_p), ("layer_sizes", C.c_void_p),
                ("weights", C.c_void_p), ("sf_shift", C.c_void_p), ("sf_scale", C.c_void_p),
                ("activation", C.c_int32), ("sf_rc", C.c_void_p)]


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build())
        L.oracle_fc.restype = C.c_double
        L.oracle_fc.argtypes = [C.c_double, C.c_double]
        L.oracle_dfc.restype = C.c_double
        L.oracle_dfc.argtypes = [C.c_double, C.c_double]
        L.oracle_wrap.restype = None
        L.oracle_wrap.argtypes = [C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p]
        L.oracle_neighbor_list.restype = C.c_int64
        L.oracle_neighbor_list.argtypes = [C.c_int64, C.c_void_p, C.c_void_p, C.c_double,
                                           C.c_void_p, C.c_void_p, C.c_int64]
        L.oracle_mlp.restype = None
        L.oracle_mlp.argtypes = [C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.oracle_centres.restype = C.c_int32
        L.oracle_centres.argtypes = [C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p,
                                     C.c_int64, C.c_void_p] + [C.c_void_p] * 3 + [C.c_int64] + [C.c_void_p] * 3
        L.oracle_centres_ex.restype = C.c_int32
        L.oracle_centres_ex.argtypes = L.oracle_centres.argtypes + [C.c_int32, C.c_void_p, C.c_void_p, C.c_int64]
        L.oracle_neighbors_of.restype = C.c_int64
        L.oracle_neighbors_of.argtypes = [C.c_int64, C.c_void_p, C.c_void_p, C.c_double, C.c_int64,
                                          C.c_void_p, C.c_int64]
        L.oracle_cells_build.restype = C.c_void_p
        L.oracle_cells_build.argtypes = [C.c_int64, C.c_void_p, C.c_void_p, C.c_double]
        L.oracle_cells_free.restype = None
        L.oracle_cells_free.argtypes = [C.c_void_p]
        L.oracle_neighbors_of_cells.restype = C.c_int64
        L.oracle_neighbors_of_cells.argtypes = [C.c_void_p, C.c_int64, C.c_void_p, C.c_int64]
        _lib = L
    return _lib


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


class OracleModel:
    """Holds the flattened model arrays alive for the C struct."""

    def __init__(self, model):
        sf = np.ascontiguousarray(model.sf)
        assert sf.dtype.itemsize == C.sizeof(_SF)
        self.sf = sf
        self.n_elem = len(model.elements)
        self.n_layers = np.array([len(ls) - 1 for ls in model.layer_sizes], dtype=np.int32)
        self.layer_sizes = np.array([s for ls in model.layer_sizes for s in ls], dtype=np.int32)
        self.weights = np.ascontiguousarray(np.concatenate(model.weights), dtype=np.float64)
        self.n_sf_per_elem = [int(np.sum(sf["central"] == e)) for e in range(self.n_elem)]
        self.g_stride = max(self.n_sf_per_elem)
        self.rc = float(model.rc)
        # model generality: optional affine SF scaling and tanh activation
        sc = getattr(model, "sf_scaling", None)
        self.sf_shift = None if sc is None else np.ascontiguousarray(np.concatenate([np.asarray(a, dtype=np.float64) for a, _ in sc]))
        self.sf_scale = None if sc is None else np.ascontiguousarray(np.concatenate([np.asarray(b, dtype=np.float64) for _, b in sc]))
        self.activation = {"softplus": 0, "tanh": 1}[getattr(model, "activation", "softplus")]
        # per-SF cutoff radii, in the order of model.sf (None: the global rc for all)
        rcs = getattr(model, "sf_cutoffs", None)
        self.sf_rc = None if rcs is None else np.ascontiguousarray(rcs, dtype=np.float64)
        assert self.sf_rc is None or (self.sf_rc.shape == (sf.shape[0],) and np.all(self.sf_rc > 0) and np.all(self.sf_rc <= self.rc))
        self.c = _Model(self.n_elem, self.rc, sf.shape[0], _ptr(sf), _ptr(self.n_layers),
                        _ptr(self.layer_sizes), _ptr(self.weights), _ptr(self.sf_shift), _ptr(self.sf_scale),
                        self.activation, _ptr(self.sf_rc))


def fc(r, rc):
    return lib().oracle_fc(float(r), float(rc))


def dfc(r, rc):
    return lib().oracle_dfc(float(r), float(rc))


def wrap(pos, box):
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    box = np.ascontiguousarray(box, dtype=np.float64)
    out = np.empty_like(pos)
    lib().oracle_wrap(pos.shape[0], _ptr(pos), _ptr(box), _ptr(out))
    return out


def neighbor_list(pos, box, rc):
    """Brute-force O(N^2) minimum-image list -> (offsets int64[N+1], idx int32[total]), rows ascending."""
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    box = np.ascontiguousarray(box, dtype=np.float64)
    n = pos.shape[0]
    off = np.zeros(n + 1, dtype=np.int64)
    total = lib().oracle_neighbor_list(n, _ptr(pos), _ptr(box), float(rc), _ptr(off), None, 0)
    idx = np.empty(max(total, 1), dtype=np.int32)
    lib().oracle_neighbor_list(n, _ptr(pos), _ptr(box), float(rc), _ptr(off), _ptr(idx), total)
    return off, idx[:total]


def neighbor_rows(pos, box, rc, atoms, search="brute"):
    """Rows N(m) (ascending original indices) of the given atoms.  search = "brute": the O(N) scan per row
    (the definition); "cells": the cell-prefiltered scan (same predicate, pinned equal to "brute")."""
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    box = np.ascontiguousarray(box, dtype=np.float64)
    n = pos.shape[0]
    w = wrap(pos, box)
    L = lib()
    buf = np.empty(max(n, 1), dtype=np.int32)
    cells = L.oracle_cells_build(n, _ptr(w), _ptr(box), float(rc)) if search == "cells" else None
    assert search in ("brute", "cells")
    rows = []
    try:
        for m in atoms:
            if cells is not None:
                cnt = L.oracle_neighbors_of_cells(cells, int(m), _ptr(buf), n)
            else:
                cnt = L.oracle_neighbors_of(n, _ptr(w), _ptr(box), float(rc), int(m), _ptr(buf), n)
            rows.append(buf[:cnt].copy())
    finally:
        if cells is not None:
            L.oracle_cells_free(cells)
    return rows


def mlp(layer_sizes, weights, G, want_beta=True):
    sizes = np.asarray(layer_sizes, dtype=np.int32)
    w = np.ascontiguousarray(weights, dtype=np.float64)
    G = np.ascontiguousarray(G, dtype=np.float64)
    e = C.c_double(0.0)
    beta = np.zeros(sizes[0], dtype=np.float64) if want_beta else None
    lib().oracle_mlp(len(sizes) - 1, _ptr(sizes), _ptr(w), _ptr(G), C.byref(e), _ptr(beta))
    return e.value, beta


class Result:
    pass


def centres(om: OracleModel, pos, types, box, sel=None, forces=True, want_g=True, search="brute", rows=False,
            F_accum=None):
    """Run the path for the selected centres (None = all atoms).

    Returns Result with e_atom[n_sel], G, dEdG [n_sel][g_stride], nbr_count[n_sel],
    F[N][3] (contributions of the selected centres only; total force if sel is None),
    e_total (sum over selected), timing (s in neighbour search, s in the rest).
    search: "brute" (the definition) or "cells" (cell-prefiltered, same rows; whole-system goldens).
    rows=True: also row_off int64[n_sel+1], row_idx int32[total]: the neighbour rows of the selected centres.
    F_accum: a float64 [N][3] array the force contributions are ADDED to (instead of a fresh zero array)."""
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    types = np.ascontiguousarray(types, dtype=np.int32)
    box = np.ascontiguousarray(box, dtype=np.float64)
    n = pos.shape[0]
    if sel is None:
        sel_a, n_sel = None, n
    else:
        sel_a = np.ascontiguousarray(sel, dtype=np.int64)
        n_sel = sel_a.shape[0]
    r = Result()
    r.e_atom = np.zeros(n_sel, dtype=np.float64)
    r.G = np.zeros((n_sel, om.g_stride), dtype=np.float64) if want_g else None
    r.dEdG = np.zeros((n_sel, om.g_stride), dtype=np.float64) if want_g else None
    r.nbr_count = np.zeros(n_sel, dtype=np.int32)
    if forces and F_accum is not None:
        assert F_accum.dtype == np.float64 and F_accum.shape == (n, 3) and F_accum.flags.c_contiguous
        r.F = F_accum
    else:
        r.F = np.zeros((n, 3), dtype=np.float64) if forces else None
    timing = np.zeros(2, dtype=np.float64)
    skind = {"brute": 0, "cells": 1}[search]
    if rows:
        cap = 256 * max(n_sel, 1)
        r.row_off = np.zeros(n_sel + 1, dtype=np.int64)
        r.row_idx = np.empty(cap, dtype=np.int32)
    else:
        cap, r.row_off, r.row_idx = 0, None, None
    rcode = lib().oracle_centres_ex(C.byref(om.c), n, _ptr(pos), _ptr(types), _ptr(box), n_sel, _ptr(sel_a),
                                    _ptr(r.e_atom), _ptr(r.G), _ptr(r.dEdG), om.g_stride,
                                    _ptr(r.nbr_count), _ptr(r.F), _ptr(timing), skind,
                                    _ptr(r.row_off), _ptr(r.row_idx), cap)
    if rows and rcode == 0:
        if r.row_off[-1] > cap:
            raise ValueError("oracle.centres(rows=True): more than 256 neighbours per centre on average")
        r.row_idx = r.row_idx[:r.row_off[-1]]
    if rcode != 0:
        raise ValueError("oracle_centres: invalid input (type out of range or box < 2 rc)")
    r.e_total = float(np.sum(r.e_atom))
    r.timing = timing
    return r


def compute(om: OracleModel, pos, types, box, forces=True):
    """Whole system: e_atom[N], e_total, F[N][3], G, dEdG."""
    return centres(om, pos, types, box, None, forces)


def forces_on(om: OracleModel, pos, types, box, atoms, offsets=None, idx=None):
    """Total force on each atom m in `atoms`: F_m = - sum_{i in N(m) + {m}} beta_i . dG_i/dr_m,
    obtained by running the path for the centres N(m) + {m} and reading row m.
    Also returns E_m, G_m.  (For sampled parity on systems too big for compute().)"""
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    types = np.ascontiguousarray(types, dtype=np.int32)
    box = np.ascontiguousarray(box, dtype=np.float64)
    n = pos.shape[0]
    w = wrap(pos, box)
    out_f, out_e, out_g, out_rows = [], [], [], []
    L = lib()
    buf = np.empty(n, dtype=np.int32)
    for m in atoms:
        cnt = L.oracle_neighbors_of(n, _ptr(w), _ptr(box), om.rc, int(m), _ptr(buf), n)
        row = buf[:cnt].copy()
        sel = np.concatenate([[int(m)], row.astype(np.int64)])
        r = centres(om, pos, types, box, sel, forces=True)
        out_f.append(r.F[int(m)].copy())
        out_e.append(r.e_atom[0])
        out_g.append(r.G[0].copy())
        out_rows.append(row)
    res = Result()
    res.F = np.array(out_f)
    res.e_atom = np.array(out_e)
    res.G = np.array(out_g)
    res.rows = out_rows
    return res
