"""Thin ctypes binding of libnnp_b200.so (C ABI: include/nnp.h).  Argument marshalling
only -- every step of the path runs in the CUDA kernels.  PyTorch is used for device
memory and streams.  There is no CPU fallback: if the library is missing or there is no
CUDA device the calls raise."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
# the in-tree build; NNP_B200_LIBRARY points at another build of the same sources (kernel-variant comparisons)
LIB_PATH = os.environ.get("NNP_B200_LIBRARY") or os.path.join(HERE, "libnnp_b200.so")

NNP_OK = 0
STATUS_NAMES = {0: "NNP_OK", 1: "NNP_ERR_INVALID_ARG", 2: "NNP_ERR_BOX_TOO_SMALL", 3: "NNP_ERR_TYPE_RANGE",
                4: "NNP_ERR_NEIGHBOR_OVERFLOW", 5: "NNP_ERR_WORKSPACE", 6: "NNP_ERR_CUDA", 7: "NNP_ERR_NONFINITE",
                8: "NNP_ERR_LIMIT", 9: "NNP_ERR_FORCE_RANGE"}
N_STAGES = 6
STAGE_NAMES = ("sort", "neighbors", "symmetry_functions", "networks", "forces", "finalize")

# every symbol include/nnp.h declares
EXPORTS = ("nnp_create", "nnp_table_kernels", "nnp_destroy", "nnp_set_max_neighbors", "nnp_workspace_bytes", "nnp_compute",
           "nnp_compute_host", "nnp_set_sf_scaling", "nnp_set_activation", "nnp_set_sf_cutoffs", "nnp_set_precision", "nnp_set_deterministic_forces", "nnp_set_neighbor_skin", "nnp_invalidate_neighbors", "nnp_get_neighbor_rebuilds", "nnp_md_run", "nnp_md_kinetic_energy", "nnp_md_kinetic_energy_noalloc", "nnp_sync_status", "nnp_get_neighbor_counts", "nnp_get_neighbors", "nnp_get_sf",
           "nnp_get_dedg", "nnp_g_stride", "nnp_set_timing", "nnp_get_timings", "nnp_last_launch_count",
           "nnp_uses_fast_path", "nnp_measure_fp64_peak", "nnp_last_error", "nnp_version")


KERNEL_NAMES = ("generic", "base12", "wide32", "free32", "free16", "multi")


def table_kernels(model):
    """Which kernels each element of `model` would run on (host only, no GPU needed) -> tuple of KERNEL_NAMES."""
    L = load_library()
    sf = np.ascontiguousarray(model.sf)
    out = np.zeros(len(model.elements), dtype=np.int32)
    st = L.nnp_table_kernels(len(model.elements), float(model.rc), int(sf.shape[0]), sf.ctypes.data_as(C.c_void_p),
                             out.ctypes.data_as(C.c_void_p))
    if st != 0:
        raise NNPError(st, L.nnp_last_error(None).decode())
    return tuple(KERNEL_NAMES[k] for k in out)


class NNPError(RuntimeError):
    def __init__(self, status, msg=""):
        self.status = status
        super().__init__("%s: %s" % (STATUS_NAMES.get(status, status), msg))


class _SF(C.Structure):
    _fields_ = [("central", C.c_int32), ("kind", C.c_int32), ("e1", C.c_int32), ("e2", C.c_int32),
                ("eta", C.c_double), ("rs", C.c_double), ("lam", C.c_double), ("zeta", C.c_double)]


_lib = None


def load_library():
    """dlopen the in-tree library (fails loudly if it has not been built)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise OSError("libnnp_b200.so is not built: run `python -c 'import __graft_entry__ as g; g.build()'` "
                      "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp, i32, i64, dbl = C.c_void_p, C.c_int32, C.c_int64, C.c_double
    L.nnp_create.restype = C.c_int
    L.nnp_create.argtypes = [C.POINTER(vp), i32, C.POINTER(C.c_char_p), dbl, i32, vp, vp, C.POINTER(vp),
                             C.POINTER(vp), i32]
    L.nnp_table_kernels.restype = C.c_int
    L.nnp_table_kernels.argtypes = [i32, dbl, i32, vp, vp]
    L.nnp_destroy.restype = None
    L.nnp_destroy.argtypes = [vp]
    L.nnp_set_max_neighbors.restype = C.c_int
    L.nnp_set_max_neighbors.argtypes = [vp, i32]
    L.nnp_workspace_bytes.restype = C.c_size_t
    L.nnp_workspace_bytes.argtypes = [vp, i64]
    L.nnp_compute.restype = C.c_int
    L.nnp_compute.argtypes = [vp, i64, vp, vp, C.POINTER(dbl), vp, vp, vp, vp, C.c_size_t, vp]
    L.nnp_compute_host.restype = C.c_int
    L.nnp_compute_host.argtypes = [vp, i64, vp, vp, C.POINTER(dbl), vp, vp, vp]
    L.nnp_set_sf_scaling.restype = C.c_int
    L.nnp_set_sf_scaling.argtypes = [vp, i32, vp, vp]
    L.nnp_set_activation.restype = C.c_int
    L.nnp_set_activation.argtypes = [vp, i32]
    L.nnp_set_sf_cutoffs.restype = C.c_int
    L.nnp_set_sf_cutoffs.argtypes = [vp, i32, vp]
    L.nnp_set_precision.restype = C.c_int
    L.nnp_set_precision.argtypes = [vp, i32]
    L.nnp_set_deterministic_forces.restype = C.c_int
    L.nnp_set_deterministic_forces.argtypes = [vp, i32]
    L.nnp_set_neighbor_skin.restype = C.c_int
    L.nnp_set_neighbor_skin.argtypes = [vp, C.c_double]
    L.nnp_invalidate_neighbors.restype = C.c_int
    L.nnp_invalidate_neighbors.argtypes = [vp]
    L.nnp_get_neighbor_rebuilds.restype = C.c_int
    L.nnp_get_neighbor_rebuilds.argtypes = [vp, vp, vp]
    L.nnp_md_run.restype = C.c_int
    L.nnp_md_run.argtypes = [vp, i32, dbl, C.POINTER(dbl), i64, vp, vp, vp, C.POINTER(dbl), vp, vp, vp, vp,
                             C.c_size_t, vp]
    L.nnp_md_kinetic_energy.restype = C.c_int
    L.nnp_md_kinetic_energy.argtypes = [vp, C.POINTER(dbl), i64, vp, vp, vp, vp, C.c_size_t, vp]
    L.nnp_md_kinetic_energy_noalloc.restype = C.c_int
    L.nnp_md_kinetic_energy_noalloc.argtypes = [vp, C.POINTER(dbl), i64, vp, vp, vp, vp]
    L.nnp_sync_status.restype = C.c_int
    L.nnp_sync_status.argtypes = [vp]
    L.nnp_get_neighbor_counts.restype = C.c_int
    L.nnp_get_neighbor_counts.argtypes = [vp, vp]
    L.nnp_get_neighbors.restype = C.c_int
    L.nnp_get_neighbors.argtypes = [vp, vp, vp, i64]
    L.nnp_get_sf.restype = C.c_int
    L.nnp_get_sf.argtypes = [vp, vp]
    L.nnp_get_dedg.restype = C.c_int
    L.nnp_get_dedg.argtypes = [vp, vp]
    L.nnp_g_stride.restype = i32
    L.nnp_g_stride.argtypes = [vp]
    L.nnp_set_timing.restype = C.c_int
    L.nnp_set_timing.argtypes = [vp, i32]
    L.nnp_get_timings.restype = C.c_int
    L.nnp_get_timings.argtypes = [vp, C.POINTER(dbl)]
    L.nnp_last_launch_count.restype = i32
    L.nnp_last_launch_count.argtypes = [vp]
    L.nnp_uses_fast_path.restype = i32
    L.nnp_uses_fast_path.argtypes = [vp]
    L.nnp_measure_fp64_peak.restype = C.c_int
    L.nnp_measure_fp64_peak.argtypes = [i32, dbl, C.POINTER(dbl), C.POINTER(dbl)]
    L.nnp_last_error.restype = C.c_char_p
    L.nnp_last_error.argtypes = [vp]
    L.nnp_version.restype = C.c_char_p
    L.nnp_version.argtypes = []
    _lib = L
    return L


def measure_fp64_peak(device: int = 0, seconds: float = 0.5):
    """-> (burst, sustained) thread-level DFMA instructions per second."""
    L = load_library()
    a, b = C.c_double(0.0), C.c_double(0.0)
    st = L.nnp_measure_fp64_peak(device, seconds, C.byref(a), C.byref(b))
    if st != NNP_OK:
        raise NNPError(st, "nnp_measure_fp64_peak")
    return a.value, b.value


class NNP:
    """nnp_create / nnp_compute with torch tensors as device buffers.

    elements: names; rc: cutoff; sf: structured array (central, kind, e1, e2, eta, rs, lam, zeta);
    layer_sizes / weights: per element (see include/nnp.h)."""

    def __init__(self, elements, rc, sf, layer_sizes, weights, device: int = 0):
        import torch  # device memory + streams only
        self._torch = torch
        self._L = load_library()
        self._h = C.c_void_p(None)
        self.device = int(device)
        sf = np.ascontiguousarray(sf)
        if sf.dtype.itemsize != C.sizeof(_SF):
            raise ValueError("sf must have 48-byte records")
        n_elem = len(elements)
        names = (C.c_char_p * n_elem)(*[str(e).encode() for e in elements])
        n_layers = np.array([len(ls) - 1 for ls in layer_sizes], dtype=np.int32)
        ls_arrays = [np.ascontiguousarray(ls, dtype=np.int32) for ls in layer_sizes]
        w_arrays = [np.ascontiguousarray(w, dtype=np.float64) for w in weights]
        ls_ptrs = (C.c_void_p * n_elem)(*[a.ctypes.data for a in ls_arrays])
        w_ptrs = (C.c_void_p * n_elem)(*[a.ctypes.data for a in w_arrays])
        st = self._L.nnp_create(C.byref(self._h), n_elem, names, float(rc), int(sf.shape[0]),
                                sf.ctypes.data_as(C.c_void_p), n_layers.ctypes.data_as(C.c_void_p),
                                ls_ptrs, w_ptrs, self.device)
        if st != NNP_OK:
            msg = self._L.nnp_last_error(None).decode()
            self._h = C.c_void_p(None)
            raise NNPError(st, msg)
        self.n_elem = n_elem
        self.rc = float(rc)
        self.g_stride = int(self._L.nnp_g_stride(self._h))
        self._ws = None
        self._ws_n = -1

    @classmethod
    def from_model(cls, model, device: int = 0):
        """model: any object with .elements .rc .sf .layer_sizes .weights (e.g. workloads.Model)."""
        obj = cls(model.elements, model.rc, model.sf, model.layer_sizes, model.weights, device)
        if getattr(model, "sf_scaling", None) is not None:
            for e, (shift, scale) in enumerate(model.sf_scaling):
                obj.set_sf_scaling(e, shift, scale)
        if getattr(model, "activation", "softplus") != "softplus":
            obj.set_activation(model.activation)
        if getattr(model, "sf_cutoffs", None) is not None:
            obj.set_sf_cutoffs(model.sf_cutoffs)
        return obj

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self._L.nnp_destroy(self._h)
            self._h = C.c_void_p(None)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, st):
        if st != NNP_OK:
            raise NNPError(st, self._L.nnp_last_error(self._h).decode())

    # ---- configuration -------------------------------------------------------------------
    def set_max_neighbors(self, k: int):
        self._check(self._L.nnp_set_max_neighbors(self._h, int(k)))
        self._ws = None
        self._ws_n = -1

    def set_timing(self, on: bool):
        self._check(self._L.nnp_set_timing(self._h, 1 if on else 0))

    def uses_fast_path(self) -> bool:
        return bool(self._L.nnp_uses_fast_path(self._h))

    def workspace_bytes(self, n_atoms: int) -> int:
        return int(self._L.nnp_workspace_bytes(self._h, int(n_atoms)))

    # ---- the hot path ----------------------------------------------------------------------
    def compute(self, pos, types, box, out=None, sync=True):
        """pos [N,3] f64 cuda tensor, types [N] i32 cuda tensor, box 3 floats (host).
        -> (e_atom [N], e_total [1], force [N,3]) cuda tensors.  Enqueued on torch's current stream."""
        torch = self._torch
        n = int(pos.shape[0])
        assert pos.is_cuda and pos.dtype == torch.float64 and pos.is_contiguous()
        assert types.is_cuda and types.dtype == torch.int32 and types.is_contiguous()
        dev = pos.device
        if self._ws is None or self._ws_n != n:
            nbytes = self.workspace_bytes(n)
            self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=dev)
            self._ws_n = n
        ws_ptr = (self._ws.data_ptr() + 255) // 256 * 256
        if out is None:
            e_atom = torch.empty(n, dtype=torch.float64, device=dev)
            e_total = torch.empty(1, dtype=torch.float64, device=dev)
            force = torch.empty((n, 3), dtype=torch.float64, device=dev)
        else:
            e_atom, e_total, force = out
        boxc = (C.c_double * 3)(*[float(b) for b in box])
        stream = torch.cuda.current_stream(dev).cuda_stream
        st = self._L.nnp_compute(self._h, n, C.c_void_p(pos.data_ptr()), C.c_void_p(types.data_ptr()), boxc,
                                 C.c_void_p(e_atom.data_ptr()), C.c_void_p(e_total.data_ptr()),
                                 C.c_void_p(force.data_ptr()), C.c_void_p(ws_ptr),
                                 self._ws.numel() - (ws_ptr - self._ws.data_ptr()), C.c_void_p(stream))
        self._check(st)
        if sync:
            self.sync_status()
        return e_atom, e_total, force

    # ---- model generality ------------------------------------------------------------
    def set_sf_scaling(self, elem, shift, scale):
        """Network input of element `elem`: x = scale * (G - shift); None, None switches it off."""
        if shift is None:
            self._check(self._L.nnp_set_sf_scaling(self._h, int(elem), None, None))
            return
        a = np.ascontiguousarray(shift, dtype=np.float64)
        b = np.ascontiguousarray(scale, dtype=np.float64)
        self._check(self._L.nnp_set_sf_scaling(self._h, int(elem), a.ctypes.data_as(C.c_void_p),
                                               b.ctypes.data_as(C.c_void_p)))

    def set_activation(self, name):
        self._check(self._L.nnp_set_activation(self._h, {"softplus": 0, "tanh": 1}[name]))

    def set_precision(self, mode):
        """"f64" (default) or "mixed" (FP32 staging and per-triplet arithmetic; include/nnp.h nnp_set_precision)."""
        self._check(self._L.nnp_set_precision(self._h, {"f64": 0, "mixed": 1}[mode]))

    def set_neighbor_skin(self, skin: float):
        """nnp_set_neighbor_skin: reuse the neighbour list across calls with a Verlet skin (Angstrom; 0 = off)."""
        self._check(self._L.nnp_set_neighbor_skin(self._h, float(skin)))
        self._ws = None            # the workspace grows by the candidate list
        self._ws_n = -1

    def invalidate_neighbors(self):
        self._check(self._L.nnp_invalidate_neighbors(self._h))

    def neighbor_rebuilds(self):
        """(calls, rebuilds) since set_neighbor_skin."""
        a, b = C.c_int64(0), C.c_int64(0)
        self._check(self._L.nnp_get_neighbor_rebuilds(self._h, C.byref(a), C.byref(b)))
        return int(a.value), int(b.value)

    def set_deterministic_forces(self, on: bool):
        """Fixed-point (2^-40 eV/A) global force accumulation: bit-reproducible forces (include/nnp.h)."""
        self._check(self._L.nnp_set_deterministic_forces(self._h, 1 if on else 0))

    def set_sf_cutoffs(self, rcs):
        """Per-SF cutoff radii in the order of the model's SF table (each <= rc); None = the global rc."""
        if rcs is None:
            self._check(self._L.nnp_set_sf_cutoffs(self._h, 0, None))
            return
        a = np.ascontiguousarray(rcs, dtype=np.float64)
        self._check(self._L.nnp_set_sf_cutoffs(self._h, int(a.shape[0]), a.ctypes.data_as(C.c_void_p)))

    # ---- MD loop around the path (velocity Verlet, NVE) ---------------------------------------------
    def _ws_ptr(self, n, dev):
        torch = self._torch
        if self._ws is None or self._ws_n != n:
            self._ws = torch.empty(self.workspace_bytes(n) + 256, dtype=torch.uint8, device=dev)
            self._ws_n = n
        ptr = (self._ws.data_ptr() + 255) // 256 * 256
        return ptr, self._ws.numel() - (ptr - self._ws.data_ptr())

    def md_run(self, n_steps, dt_fs, masses, pos, vel, types, box, state, sync=True):
        """n_steps velocity-Verlet steps in place on pos / vel (cuda f64 [N,3]); `state` = (e_atom, e_total,
        force) from a compute() of pos (the forces are read on entry, everything is updated)."""
        n = int(pos.shape[0])
        e_atom, e_total, force = state
        ws_ptr, ws_len = self._ws_ptr(n, pos.device)
        m = (C.c_double * len(masses))(*[float(x) for x in masses])
        boxc = (C.c_double * 3)(*[float(b) for b in box])
        stream = self._torch.cuda.current_stream(pos.device).cuda_stream
        st = self._L.nnp_md_run(self._h, int(n_steps), float(dt_fs), m, n, C.c_void_p(pos.data_ptr()),
                                C.c_void_p(vel.data_ptr()), C.c_void_p(types.data_ptr()), boxc,
                                C.c_void_p(e_atom.data_ptr()), C.c_void_p(e_total.data_ptr()),
                                C.c_void_p(force.data_ptr()), C.c_void_p(ws_ptr), ws_len, C.c_void_p(stream))
        self._check(st)
        if sync:
            self.sync_status()

    def kinetic_energy(self, masses, vel, types):
        """sum m v^2 / 2 in eV -> cuda f64 [1]."""
        n = int(vel.shape[0])
        out = self._torch.empty(1, dtype=self._torch.float64, device=vel.device)
        ws_ptr, ws_len = self._ws_ptr(n, vel.device)
        m = (C.c_double * len(masses))(*[float(x) for x in masses])
        stream = self._torch.cuda.current_stream(vel.device).cuda_stream
        self._check(self._L.nnp_md_kinetic_energy(self._h, m, n, C.c_void_p(vel.data_ptr()),
                                                  C.c_void_p(types.data_ptr()), C.c_void_p(out.data_ptr()),
                                                  C.c_void_p(ws_ptr), ws_len, C.c_void_p(stream)))
        return out

    def kinetic_energy_noalloc(self, masses, vel, types, out, n_atoms=None):
        """nnp_md_kinetic_energy_noalloc: the same sum with no workspace and no allocation inside the library; the caller
        owns `out` (cuda f64 [1]).  n_atoms <= 4,194,304; calls that overlap on the GPU race on the library's static scratch."""
        n = int(vel.shape[0]) if n_atoms is None else int(n_atoms)
        m = (C.c_double * len(masses))(*[float(x) for x in masses])
        stream = self._torch.cuda.current_stream(vel.device).cuda_stream
        self._check(self._L.nnp_md_kinetic_energy_noalloc(self._h, m, n, C.c_void_p(vel.data_ptr()),
                                                          C.c_void_p(types.data_ptr()), C.c_void_p(out.data_ptr()),
                                                          C.c_void_p(stream)))
        return out

    def compute_host(self, pos, types, box, out=None):
        """Same evaluation with HOST numpy / pinned-torch buffers (copies inside the call)."""
        def ptr(a):
            return C.c_void_p(a.data_ptr()) if hasattr(a, "data_ptr") else a.ctypes.data_as(C.c_void_p)
        n = int(pos.shape[0])
        if out is None:
            e_atom = np.empty(n, dtype=np.float64)
            e_total = np.empty(1, dtype=np.float64)
            force = np.empty((n, 3), dtype=np.float64)
        else:
            e_atom, e_total, force = out
        boxc = (C.c_double * 3)(*[float(b) for b in box])
        st = self._L.nnp_compute_host(self._h, n, ptr(pos), ptr(types), boxc, ptr(e_atom), ptr(e_total), ptr(force))
        self._check(st)
        return e_atom, e_total, force

    def sync_status(self):
        self._check(self._L.nnp_sync_status(self._h))

    def last_launch_count(self) -> int:
        return int(self._L.nnp_last_launch_count(self._h))

    def timings_ms(self):
        ms = (C.c_double * N_STAGES)()
        self._check(self._L.nnp_get_timings(self._h, ms))
        return dict(zip(STAGE_NAMES, [float(x) for x in ms]))

    # ---- debug / parity exports of the last compute ----------------------------------------------
    def neighbors(self, n_atoms: int):
        """-> (offsets int64[N+1], idx int32[total]) cuda tensors; caller's atom ids, rows ascending."""
        torch = self._torch
        dev = torch.device("cuda", self.device)
        off = torch.empty(n_atoms + 1, dtype=torch.int64, device=dev)
        self._check(self._L.nnp_get_neighbors(self._h, C.c_void_p(off.data_ptr()), None, 0))
        total = int(off[-1].item()) if n_atoms > 0 else 0
        idx = torch.empty(max(total, 1), dtype=torch.int32, device=dev)
        self._check(self._L.nnp_get_neighbors(self._h, C.c_void_p(off.data_ptr()), C.c_void_p(idx.data_ptr()), total))
        return off, idx[:total]

    def neighbor_counts(self, n_atoms: int):
        torch = self._torch
        c = torch.empty(max(n_atoms, 1), dtype=torch.int32, device=torch.device("cuda", self.device))
        self._check(self._L.nnp_get_neighbor_counts(self._h, C.c_void_p(c.data_ptr())))
        return c[:n_atoms]

    def symmetry_functions(self, n_atoms: int):
        torch = self._torch
        g = torch.empty((max(n_atoms, 1), self.g_stride), dtype=torch.float64, device=torch.device("cuda", self.device))
        self._check(self._L.nnp_get_sf(self._h, C.c_void_p(g.data_ptr())))
        return g[:n_atoms]

    def dedg(self, n_atoms: int):
        torch = self._torch
        g = torch.empty((max(n_atoms, 1), self.g_stride), dtype=torch.float64, device=torch.device("cuda", self.device))
        self._check(self._L.nnp_get_dedg(self._h, C.c_void_p(g.data_ptr())))
        return g[:n_atoms]
