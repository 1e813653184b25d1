"""ctypes binding of include/npfem.h - same names, argument marshalling only.

PyTorch supplies device memory (the workspace and the user buffers are torch tensors) and the
CUDA stream; every arithmetic step runs in libnpfem_b200.so.  If the library is missing or has
no CUDA device the calls raise: there is no CPU fallback.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

NPFEM_F32, NPFEM_F64 = 32, 64
NPFEM_DEVICE, NPFEM_HOST = 0, 1
OPT_DIAGNOSTICS, OPT_GLOBAL_STEP_MATH, OPT_LOCAL_STEP_IMPL, OPT_KERNEL_TIMING, OPT_UPDATE_MODE = 1, 2, 3, 4, 5
OPT_FORCE_MEDIAN_FILTER = 6
OPT_FUSED_STEP = 7
KIND_NAMES = ("prologue", "local", "global", "epilogue", "line_search", "fused_step", "global_simt")
FEATURE_DIAGNOSTICS, FEATURE_LINE_SEARCH, FEATURE_COLLISIONS = 1, 2, 4
_ERR_NAMES = {-1: "NPFEM_EINVAL", -2: "NPFEM_EMESH", -3: "NPFEM_ECUDA", -4: "NPFEM_ENOMEM", -5: "NPFEM_ESTATE"}

EXPORTED_SYMBOLS = (
    "npfem_create", "npfem_workspace_bytes", "npfem_bind_workspace", "npfem_scratch_bytes", "npfem_bind_scratch", "npfem_set_option",
    "npfem_set_state", "npfem_set_forces", "npfem_step", "npfem_step_host", "npfem_get_state", "npfem_get_objective",
    "npfem_get_kernel_times", "npfem_launch_count", "npfem_last_error", "npfem_version", "npfem_destroy",
    "npfem_local_schedule_stats", "npfem_set_line_search", "npfem_get_step_lengths", "npfem_set_velocity_cap", "npfem_set_collisions",
    "npfem_clear_collisions", "npfem_probe_fma_peak",
    "npfem_quad_schedule_stats", "npfem_quadmp_schedule_stats", "npfem_invert_spd_tmp_bytes", "npfem_invert_spd", "npfem_invert_spd_static", "npfem_invert_spd_last_error",
)


class NpfemError(RuntimeError):
    def __init__(self, code: int, message: str):
        super().__init__(f"{_ERR_NAMES.get(code, code)}: {message}")
        self.code = code


class _Material(C.Structure):
    _fields_ = [(k, C.c_double) for k in (
        "skalak_B", "skalak_C", "skalak_D", "k_bending", "k_volume", "rayleigh_alpha", "rayleigh_beta",
        "kappa_damping", "density")]


class _CellType(C.Structure):
    _fields_ = [("n_vertices", C.c_int32), ("n_triangles", C.c_int32),
                ("rest_positions", C.POINTER(C.c_double)), ("triangles", C.POINTER(C.c_int32)),
                ("material", _Material)]


def library_path() -> str:
    return os.path.join(os.path.dirname(os.path.abspath(__file__)), "lib", "libnpfem_b200.so")


_LIB = None


def load_library(build_if_missing: bool = True) -> C.CDLL:
    """dlopen the in-tree library (building it with nvcc first if it is absent)."""
    global _LIB
    if _LIB is not None:
        return _LIB
    path = library_path()
    if not os.path.exists(path):
        if not build_if_missing:
            raise FileNotFoundError(f"{path} is missing: run `python -m paper_1911_03062_b200.build`")
        from .build import build
        build()
    lib = C.CDLL(path)
    vp, i32, i64, sz = C.c_void_p, C.c_int32, C.c_int64, C.c_size_t
    lib.npfem_create.argtypes = [C.POINTER(vp), C.POINTER(_CellType), i32, C.POINTER(i32), i64, C.c_double, i32, i32, vp]
    lib.npfem_create.restype = C.c_int
    lib.npfem_workspace_bytes.argtypes = [vp]
    lib.npfem_workspace_bytes.restype = sz
    lib.npfem_bind_workspace.argtypes = [vp, vp, sz]
    lib.npfem_bind_workspace.restype = C.c_int
    lib.npfem_scratch_bytes.argtypes = [vp, i32]
    lib.npfem_scratch_bytes.restype = sz
    lib.npfem_bind_scratch.argtypes = [vp, vp, sz, i32]
    lib.npfem_bind_scratch.restype = C.c_int
    lib.npfem_set_option.argtypes = [vp, i32, i64]
    lib.npfem_set_option.restype = C.c_int
    lib.npfem_set_state.argtypes = [vp, C.POINTER(i64), i64, vp, vp, i32, i32]
    lib.npfem_set_state.restype = C.c_int
    lib.npfem_set_forces.argtypes = [vp, C.POINTER(i64), i64, vp, i32, i32]
    lib.npfem_set_forces.restype = C.c_int
    lib.npfem_step.argtypes = [vp, i32]
    lib.npfem_step.restype = C.c_int
    lib.npfem_step_host.argtypes = [vp, vp, i32, vp, vp, i32, i32]
    lib.npfem_step_host.restype = C.c_int
    lib.npfem_get_state.argtypes = [vp, C.POINTER(i64), i64, vp, vp, i32, i32]
    lib.npfem_get_state.restype = C.c_int
    lib.npfem_get_objective.argtypes = [vp, vp, i32, C.POINTER(i32), vp, i32]
    lib.npfem_get_objective.restype = C.c_int
    lib.npfem_get_kernel_times.argtypes = [vp, vp, vp, i32]
    lib.npfem_get_kernel_times.restype = C.c_int
    lib.npfem_launch_count.argtypes = [vp]
    lib.npfem_launch_count.restype = i64
    lib.npfem_last_error.argtypes = [vp]
    lib.npfem_last_error.restype = C.c_char_p
    lib.npfem_version.argtypes = []
    lib.npfem_version.restype = C.c_char_p
    lib.npfem_destroy.argtypes = [vp]
    lib.npfem_destroy.restype = None
    lib.npfem_set_line_search.argtypes = [vp, i32, C.c_double, C.c_double]
    lib.npfem_set_line_search.restype = C.c_int
    lib.npfem_set_collisions.argtypes = [vp, C.POINTER(i64), i64, vp, vp, i32, i32]
    lib.npfem_set_collisions.restype = C.c_int
    lib.npfem_clear_collisions.argtypes = [vp]
    lib.npfem_clear_collisions.restype = C.c_int
    lib.npfem_set_velocity_cap.argtypes = [vp, C.c_double]
    lib.npfem_set_velocity_cap.restype = C.c_int
    lib.npfem_get_step_lengths.argtypes = [vp, vp]
    lib.npfem_get_step_lengths.restype = C.c_int
    lib.npfem_local_schedule_stats.argtypes = [C.POINTER(_CellType), C.c_double, C.POINTER(C.c_double), i32]
    lib.npfem_local_schedule_stats.restype = C.c_int
    lib.npfem_quad_schedule_stats.argtypes = [C.POINTER(_CellType), C.c_double, C.POINTER(C.c_double), i32]
    lib.npfem_quad_schedule_stats.restype = C.c_int
    lib.npfem_quadmp_schedule_stats.argtypes = [C.POINTER(_CellType), C.c_double, C.POINTER(C.c_double), i32]
    lib.npfem_quadmp_schedule_stats.restype = C.c_int
    lib.npfem_probe_fma_peak.argtypes = [vp, i32, i32, i32, vp, C.POINTER(C.c_double)]
    lib.npfem_probe_fma_peak.restype = C.c_int
    lib.npfem_invert_spd_tmp_bytes.argtypes = [i32]
    lib.npfem_invert_spd_tmp_bytes.restype = sz
    lib.npfem_invert_spd.argtypes = [vp, vp, i32, vp, sz, vp, C.POINTER(C.c_double)]
    lib.npfem_invert_spd.restype = C.c_int
    lib.npfem_invert_spd_static.argtypes = [vp, vp, i32, vp, C.POINTER(C.c_double)]
    lib.npfem_invert_spd_static.restype = C.c_int
    lib.npfem_invert_spd_last_error.argtypes = []
    lib.npfem_invert_spd_last_error.restype = C.c_char_p
    _LIB = lib
    return lib


def _material_struct(m) -> _Material:
    return _Material(m.skalak_B, m.skalak_C, m.skalak_D, m.k_bending, m.k_volume, m.rayleigh_alpha,
                     m.rayleigh_beta, m.kappa_damping, m.density)


SCHEDULE_STAT_NAMES = ("valid", "threads", "triangles_per_thread", "wavefronts_vertex_gather",
                       "wavefronts_normal_gather", "worst_corner_store", "worst_corner_gather", "tables_consistent",
                       "smem_bytes", "build_ms")


def local_schedule_stats(cell_type, dt: float) -> dict:
    """npfem_local_schedule_stats (host-only, no GPU needed): the create-time shared-memory schedule
    of the scheduled fp32 local step for one cell type, checked by the library itself."""
    lib = load_library()
    rest = np.ascontiguousarray(cell_type.rest_positions, dtype=np.float64)
    tri = np.ascontiguousarray(cell_type.triangles, dtype=np.int32)
    ct = _CellType(rest.shape[0], tri.shape[0], rest.ctypes.data_as(C.POINTER(C.c_double)),
                   tri.ctypes.data_as(C.POINTER(C.c_int32)), _material_struct(cell_type.material))
    out = (C.c_double * len(SCHEDULE_STAT_NAMES))()
    rc = lib.npfem_local_schedule_stats(C.byref(ct), float(dt), out, len(SCHEDULE_STAT_NAMES))
    if rc != 0:
        raise NpfemError(rc, lib.npfem_last_error(None).decode())
    return dict(zip(SCHEDULE_STAT_NAMES, [float(v) for v in out]))


QUAD_STAT_NAMES = ("valid", "threads", "reads_per_vertex", "wf_vertex_gather", "wf_normal_gather", "worst_store_quarter",
                   "worst_gather_quarter", "consistent", "smem_bytes", "build_ms")


def quad_schedule_stats(cell_type, dt: float, multipass: bool = False) -> dict:
    """npfem_quad_schedule_stats / npfem_quadmp_schedule_stats (host-only): the create-time schedule of the quad local
    step (multipass: of its multi-pass variant; "threads" is then the number of passes), decoded and checked against
    the mesh by the library."""
    lib = load_library()
    rest = np.ascontiguousarray(cell_type.rest_positions, dtype=np.float64)
    tri = np.ascontiguousarray(cell_type.triangles, dtype=np.int32)
    ct = _CellType(rest.shape[0], tri.shape[0], rest.ctypes.data_as(C.POINTER(C.c_double)),
                   tri.ctypes.data_as(C.POINTER(C.c_int32)), _material_struct(cell_type.material))
    out = (C.c_double * len(QUAD_STAT_NAMES))()
    fn = lib.npfem_quadmp_schedule_stats if multipass else lib.npfem_quad_schedule_stats
    rc = fn(C.byref(ct), float(dt), out, len(QUAD_STAT_NAMES))
    if rc != 0:
        raise NpfemError(rc, lib.npfem_last_error(None).decode())
    return dict(zip(QUAD_STAT_NAMES, [float(v) for v in out]))


INVERT_STATIC_MAX_N = 258        # NPFEM_INVERT_STATIC_MAX_N of include/npfem.h


def invert_spd(H, out=None, tmp=None, stream=None):
    """npfem_invert_spd: fp64 inverse of the SPD matrix H (torch CUDA tensor [n][n], float64, contiguous) with
    caller-owned scratch `tmp` (torch uint8 CUDA tensor of >= npfem_invert_spd_tmp_bytes(n); torch allocates one if
    None).  Returns (inverse, residual).  Argument marshalling only."""
    import torch
    lib = load_library()
    n = _check_square_f64(H)
    out = torch.empty_like(H) if out is None else out
    need = lib.npfem_invert_spd_tmp_bytes(n)
    tmp = torch.empty(need, dtype=torch.uint8, device=H.device) if tmp is None else tmp
    res = C.c_double(0.0)
    st = torch.cuda.current_stream(H.device) if stream is None else stream
    rc = lib.npfem_invert_spd(C.c_void_p(H.data_ptr()), C.c_void_p(out.data_ptr()), n, C.c_void_p(tmp.data_ptr()), tmp.numel(),
                              C.c_void_p(st.cuda_stream), C.byref(res))
    if rc != 0:
        raise NpfemError(rc, lib.npfem_invert_spd_last_error().decode())
    return out, res.value


def invert_spd_static(H, out, stream=None):
    """npfem_invert_spd_static: the same inverse with the library's static device scratch (n <= INVERT_STATIC_MAX_N):
    no device allocation on this path, `out` is the caller's.  Returns the residual.  Calls that overlap on the GPU
    race on the shared scratch."""
    import torch
    lib = load_library()
    n = _check_square_f64(H)
    _check_square_f64(out)
    res = C.c_double(0.0)
    st = torch.cuda.current_stream(H.device) if stream is None else stream
    rc = lib.npfem_invert_spd_static(C.c_void_p(H.data_ptr()), C.c_void_p(out.data_ptr()), n, C.c_void_p(st.cuda_stream),
                                     C.byref(res))
    if rc != 0:
        raise NpfemError(rc, lib.npfem_invert_spd_last_error().decode())
    return res.value


def _check_square_f64(H) -> int:
    import torch
    if not (H.is_cuda and H.dtype == torch.float64 and H.dim() == 2 and H.shape[0] == H.shape[1] and H.is_contiguous()):
        raise ValueError("expected a contiguous float64 CUDA tensor [n][n]")
    return int(H.shape[0])


class Solver:
    """npfem_create / set_state / set_forces / step / get_state around one npfem_ctx.

    cell_types: objects with rest_positions [n,3] float64, triangles [T,3] int32 and a material
    carrying the npfem_material fields (e.g. workloads.CellType).  Buffers handed to set_*/get_*
    are flat: the listed cells back to back, each `[n][3]`; torch CUDA tensors are used in
    place (NPFEM_DEVICE), torch CPU tensors / numpy arrays go through the HOST path.
    """

    def __init__(self, cell_types, type_of_cell, dt: float, precision: str = "fp32", device: int = 0,
                 bind_torch_workspace: bool = True):
        import torch
        self._torch = torch
        self._lib = load_library()
        self.precision = {"fp32": NPFEM_F32, "fp64": NPFEM_F64, 32: NPFEM_F32, 64: NPFEM_F64}[precision]
        self.device = int(device)
        self.n_types = len(cell_types)
        self.type_of_cell = np.ascontiguousarray(type_of_cell, dtype=np.int32)
        self.n_cells = int(self.type_of_cell.shape[0])
        self.n_vertices = np.array([int(ct.rest_positions.shape[0]) for ct in cell_types], dtype=np.int64)
        self.total_vertices = int(self.n_vertices[self.type_of_cell].sum()) if self.n_cells else 0
        keep = []
        arr = (_CellType * self.n_types)()
        for i, ct in enumerate(cell_types):
            rest = np.ascontiguousarray(ct.rest_positions, dtype=np.float64)
            tri = np.ascontiguousarray(ct.triangles, dtype=np.int32)
            keep += [rest, tri]
            arr[i] = _CellType(rest.shape[0], tri.shape[0], rest.ctypes.data_as(C.POINTER(C.c_double)),
                               tri.ctypes.data_as(C.POINTER(C.c_int32)), _material_struct(ct.material))
        if not torch.cuda.is_available():
            raise NpfemError(-3, "no CUDA device: libnpfem_b200 has no CPU fallback")
        torch.cuda.set_device(self.device)
        self._stream = torch.cuda.current_stream(self.device)
        ctx = C.c_void_p()
        rc = self._lib.npfem_create(C.byref(ctx), arr, self.n_types,
                                    self.type_of_cell.ctypes.data_as(C.POINTER(C.c_int32)), self.n_cells,
                                    float(dt), self.precision, self.device, C.c_void_p(self._stream.cuda_stream))
        if rc != 0:
            raise NpfemError(rc, self._lib.npfem_last_error(None).decode())
        self._ctx = ctx
        self._workspace = None
        self._scratch = {}            # feature bit -> torch tensor (the caller owns the device memory, npfem.h)
        if bind_torch_workspace:
            nbytes = int(self._lib.npfem_workspace_bytes(self._ctx))
            self._workspace = torch.empty(max(nbytes, 256), dtype=torch.uint8, device=f"cuda:{self.device}")
            self._check(self._lib.npfem_bind_workspace(self._ctx, C.c_void_p(self._workspace.data_ptr()),
                                                       self._workspace.numel()))

    # ---- helpers ------------------------------------------------------------------------------
    def _check(self, rc: int) -> None:
        if rc != 0:
            raise NpfemError(rc, self._lib.npfem_last_error(self._ctx).decode())

    def _ids(self, cell_ids):
        if cell_ids is None:
            return None, 0, None
        ids = np.ascontiguousarray(cell_ids, dtype=np.int64)
        return ids.ctypes.data_as(C.POINTER(C.c_int64)), int(ids.shape[0]), ids

    def _count(self, ids) -> int:
        return 3 * (self.total_vertices if ids is None else int(self.n_vertices[self.type_of_cell[ids]].sum()))

    def _buffer(self, buf, count: int, name: str):
        """-> (pointer, dtype code, where, keepalive)"""
        torch = self._torch
        if buf is None:
            return None, None, None, None
        if isinstance(buf, torch.Tensor):
            if buf.dtype not in (torch.float32, torch.float64):
                raise TypeError(f"{name} must be float32 or float64")
            if not buf.is_contiguous() or buf.numel() != count:
                raise ValueError(f"{name} must be contiguous with {count} elements, got {buf.numel()}")
            code = NPFEM_F32 if buf.dtype == torch.float32 else NPFEM_F64
            where = NPFEM_DEVICE if buf.is_cuda else NPFEM_HOST
            return C.c_void_p(buf.data_ptr()), code, where, buf
        arr = np.asarray(buf)
        if arr.dtype not in (np.float32, np.float64):
            raise TypeError(f"{name} must be float32 or float64")
        if not arr.flags.c_contiguous or arr.size != count:
            raise ValueError(f"{name} must be C-contiguous with {count} elements, got {arr.size}")
        return C.c_void_p(arr.ctypes.data), NPFEM_F32 if arr.dtype == np.float32 else NPFEM_F64, NPFEM_HOST, arr

    def _ensure_scratch(self, feature: int) -> None:
        """With a torch-owned workspace the optional features get torch-owned scratch too (npfem_bind_scratch),
        bound before the call that enables the feature; a library-owned workspace allocates its own."""
        if self._workspace is None or feature in self._scratch:
            return
        nbytes = int(self._lib.npfem_scratch_bytes(self._ctx, feature))
        buf = self._torch.empty(max(nbytes, 256), dtype=self._torch.uint8, device=f"cuda:{self.device}")
        self._check(self._lib.npfem_bind_scratch(self._ctx, C.c_void_p(buf.data_ptr()), buf.numel(), feature))
        self._scratch[feature] = buf

    @property
    def scratch_bytes(self) -> int:
        return sum(int(b.numel()) for b in self._scratch.values())

    # ---- the C-ABI calls ----------------------------------------------------------------------
    def set_option(self, option: int, value: int) -> None:
        if option == OPT_DIAGNOSTICS and value:
            self._ensure_scratch(FEATURE_DIAGNOSTICS)
        self._check(self._lib.npfem_set_option(self._ctx, option, int(value)))

    def set_state(self, positions, velocities=None, cell_ids=None) -> None:
        ids_p, n_ids, ids = self._ids(cell_ids)
        count = self._count(ids)
        p, code, where, _k1 = self._buffer(positions, count, "positions")
        v, vcode, vwhere, _k2 = self._buffer(velocities, count, "velocities")
        if v is not None and (vcode != code or vwhere != where):
            raise ValueError("positions and velocities must share dtype and location")
        self._check(self._lib.npfem_set_state(self._ctx, ids_p, n_ids, p, v, code, where))

    def set_forces(self, forces, cell_ids=None) -> None:
        ids_p, n_ids, ids = self._ids(cell_ids)
        p, code, where, _k = self._buffer(forces, self._count(ids), "forces")
        self._check(self._lib.npfem_set_forces(self._ctx, ids_p, n_ids, p, code, where))

    def set_collisions(self, targets, stiffness, cell_ids=None) -> None:
        """PIK collision term: targets `[n][3]` and stiffness `[n]` per listed cell (same dtype and place)."""
        ids_p, n_ids, ids = self._ids(cell_ids)
        count = self._count(ids)
        p, code, where, _k = self._buffer(targets, count, "targets")
        q, code_q, where_q, _k2 = self._buffer(stiffness, count // 3, "stiffness")
        if code != code_q or where != where_q:
            raise ValueError("targets and stiffness must share dtype and location")
        self._ensure_scratch(FEATURE_COLLISIONS)
        self._check(self._lib.npfem_set_collisions(self._ctx, ids_p, n_ids, p, q, code, where))

    def clear_collisions(self) -> None:
        self._check(self._lib.npfem_clear_collisions(self._ctx))

    def step(self, n_iterations: int) -> None:
        self._check(self._lib.npfem_step(self._ctx, int(n_iterations)))

    def step_host(self, forces, n_iterations: int, positions, velocities, n_chunks: int = 0) -> None:
        """npfem_step_host: forces in, one step, {x, v} out with HOST buffers, pipelined over chunks of cells."""
        count = 3 * self.total_vertices
        f, code, where, _k0 = self._buffer(forces, count, "forces")
        p, pcode, pwhere, _k1 = self._buffer(positions, count, "positions")
        v, vcode, vwhere, _k2 = self._buffer(velocities, count, "velocities")
        if {where, pwhere, vwhere} != {NPFEM_HOST} or not (code == pcode == vcode):
            raise ValueError("step_host takes host buffers of one dtype")
        self._check(self._lib.npfem_step_host(self._ctx, f, int(n_iterations), p, v, code, int(n_chunks)))

    def get_state(self, cell_ids=None, dtype="fp64", where="device", positions=None, velocities=None):
        """Returns (positions, velocities) as flat tensors (device) or numpy arrays (host)."""
        torch = self._torch
        ids_p, n_ids, ids = self._ids(cell_ids)
        count = self._count(ids)
        if positions is None:
            if where == "device":
                tdt = torch.float32 if dtype in ("fp32", 32) else torch.float64
                positions = torch.empty(count, dtype=tdt, device=f"cuda:{self.device}")
                velocities = torch.empty_like(positions)
            else:
                ndt = np.float32 if dtype in ("fp32", 32) else np.float64
                positions = np.empty(count, dtype=ndt)
                velocities = np.empty(count, dtype=ndt)
        p, code, loc, _k1 = self._buffer(positions, count, "positions")
        v, _, _, _k2 = self._buffer(velocities, count, "velocities")
        self._check(self._lib.npfem_get_state(self._ctx, ids_p, n_ids, p, v, code, loc))
        return positions, velocities

    def get_objective(self):
        """(history [n_entries, n_cells] float64 numpy, monotone [n_cells] int32 numpy)."""
        n_entries = C.c_int32(0)
        hist = np.empty((257, max(self.n_cells, 1)), dtype=np.float64)
        mono = np.empty(max(self.n_cells, 1), dtype=np.int32)
        self._check(self._lib.npfem_get_objective(self._ctx, C.c_void_p(hist.ctypes.data), 257, C.byref(n_entries),
                                                  C.c_void_p(mono.ctypes.data), NPFEM_HOST))
        return hist[:n_entries.value, :self.n_cells].copy(), mono[:self.n_cells].copy()

    def set_line_search(self, max_halvings: int, armijo_c1: float = 1e-4, grad_tol: float = 0.0) -> None:
        """Armijo backtracking + gradient-norm stopping test for the following steps (0 = off)."""
        if max_halvings > 0:
            self._ensure_scratch(FEATURE_LINE_SEARCH)
        self._check(self._lib.npfem_set_line_search(self._ctx, int(max_halvings), float(armijo_c1), float(grad_tol)))

    def set_velocity_cap(self, v_max: float) -> None:
        """Clamp |v_{n+1}| of every vertex to v_max after each step (0 = off)."""
        self._check(self._lib.npfem_set_velocity_cap(self._ctx, float(v_max)))

    def get_step_lengths(self) -> np.ndarray:
        """alpha of the last iteration of the last step, [n_cells] in cell-id order."""
        out = np.zeros(self.n_cells, dtype=np.float64)
        self._check(self._lib.npfem_get_step_lengths(self._ctx, C.c_void_p(out.ctypes.data)))
        return out

    def get_kernel_times(self, reset: bool = True):
        """{kind: [(ms, launches) per cell type]} accumulated since the last reset (OPT_KERNEL_TIMING)."""
        ms = np.zeros((len(KIND_NAMES), self.n_types), dtype=np.float64)
        cnt = np.zeros((len(KIND_NAMES), self.n_types), dtype=np.int64)
        self._check(self._lib.npfem_get_kernel_times(self._ctx, C.c_void_p(ms.ctypes.data),
                                                     C.c_void_p(cnt.ctypes.data), 1 if reset else 0))
        return {k: [(float(ms[i, t]), int(cnt[i, t])) for t in range(self.n_types)]
                for i, k in enumerate(KIND_NAMES)}

    @property
    def launch_count(self) -> int:
        return int(self._lib.npfem_launch_count(self._ctx))

    @property
    def workspace_bytes(self) -> int:
        return int(self._lib.npfem_workspace_bytes(self._ctx))

    def close(self) -> None:
        if getattr(self, "_ctx", None):
            self._lib.npfem_destroy(self._ctx)
            self._ctx = None
            self._workspace = None
            self._scratch = {}

    def __del__(self):  # pragma: no cover
        try:
            self.close()
        except Exception:
            pass
