"""ctypes binding of include/bh.h -- argument marshalling only; every step of the path runs in the CUDA library.

PyTorch is used for device memory (the workspace tensor) and streams.  There is no CPU fallback: constructing a
``BarnesHut`` without the compiled library or without a CUDA device raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libbh_b200.so")

BH_OK = 0
STATUS = {0: "BH_OK", -1: "BH_ERR_INVALID_ARG", -2: "BH_ERR_WORKSPACE", -3: "BH_ERR_STATE", -4: "BH_ERR_CUDA",
          -5: "BH_ERR_NONFINITE", -6: "BH_ERR_CAPACITY", -7: "BH_ERR_TOO_LARGE"}

# every symbol include/bh.h declares (checked by tests/test_abi.py)
SYMBOLS = ["bh_workspace_bytes", "bh_create", "bh_destroy", "bh_set_particles", "bh_bind_particles", "bh_land_particles", "bh_get_particles", "bh_tree_build",
           "bh_compute_forces", "bh_refresh_moments", "bh_compute_forces_active", "bh_refresh_moments_active", "bh_block_init", "bh_block_step",
           "bh_block_state", "bh_set_mac", "bh_leapfrog_step", "bh_step_graph_build",
           "bh_step_graph_launch", "bh_kick_drift", "bh_sync_status", "bh_export_tree", "bh_set_stage_timing",
           "bh_get_stage_ms", "bh_get_walk_timeline", "bh_direct_forces", "bh_domain_box_static", "bh_domain_box_static_max_n", "bh_probe_fp32", "bh_last_cuda_error",
           "bh_status_string"]


class BhConfig(C.Structure):
    _fields_ = [("nleaf", C.c_int32), ("ncrit", C.c_int32), ("max_cells", C.c_int64), ("list_entries", C.c_int64),
                ("walk_mode", C.c_int32), ("walk_waves", C.c_int32), ("front_mode", C.c_int32), ("walk_private", C.c_int32)]


class BhStats(C.Structure):
    _fields_ = [("status", C.c_int32), ("n_levels", C.c_int32), ("n", C.c_int64), ("n_cells", C.c_int64),
                ("n_groups", C.c_int64), ("sum_pc", C.c_int64), ("sum_pp", C.c_int64), ("sum_mac", C.c_int64),
                ("launches", C.c_int64), ("lo", C.c_float * 3), ("hi", C.c_float * 3), ("domain_exp", C.c_int32),
                ("sort_retries", C.c_int32), ("sort_passes", C.c_int32), ("reserved", C.c_int32)]


class BhDomainBox(C.Structure):
    _fields_ = [("lo", C.c_float * 3), ("hi", C.c_float * 3), ("domain_exp", C.c_int32), ("status", C.c_int32)]


class BhBlockConfig(C.Structure):
    _fields_ = [("len_scale", C.c_float), ("eta", C.c_float), ("dt_max", C.c_float), ("max_rung", C.c_int32)]


class BhBlockStats(C.Structure):
    _fields_ = [("steps", C.c_int64), ("steps_since_rebuild", C.c_int64), ("now_tick", C.c_int64), ("n_active", C.c_int64),
                ("interactions_now", C.c_int64), ("interactions_first", C.c_int64)]


_VIEW_FIELDS = ["pos_mass", "vel", "acc_pot", "id", "key", "perm", "level_offset", "cell_level", "cell_prefix",
                "cell_pbegin", "cell_pcount", "cell_child_begin", "cell_nchild", "cell_parent", "cell_mom64", "cell_box",
                "cell_mom32", "cell_r2open", "cell_trec", "cell_erec", "group_begin", "group_cell", "group_npc", "group_npp"]


class BhTreeView(C.Structure):
    _fields_ = [(name, C.c_void_p) for name in _VIEW_FIELDS]


class BhError(RuntimeError):
    def __init__(self, code: int, what: str = ""):
        self.code = code
        super().__init__(f"{STATUS.get(code, code)} {what}".strip())


_lib = None


def load_library():
    """Load libbh_b200.so (built by paper_1106_1900_b200/build.py).  Raises if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise FileNotFoundError(f"{LIB_PATH} not built: run `python -c 'import __graft_entry__ as g; g.build()'`")
    lib = C.CDLL(LIB_PATH)
    lib.bh_workspace_bytes.restype = C.c_size_t
    lib.bh_workspace_bytes.argtypes = [C.c_int64, C.POINTER(BhConfig)]
    lib.bh_create.argtypes = [C.POINTER(C.c_void_p), C.c_int64, C.POINTER(BhConfig), C.c_void_p, C.c_size_t]
    lib.bh_destroy.argtypes = [C.c_void_p]
    lib.bh_set_particles.argtypes = [C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    lib.bh_bind_particles.argtypes = [C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    lib.bh_bind_particles.restype = C.c_int
    lib.bh_land_particles.argtypes = [C.c_void_p, C.c_void_p]
    lib.bh_land_particles.restype = C.c_int
    lib.bh_get_particles.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    lib.bh_tree_build.argtypes = [C.c_void_p, C.c_void_p]
    lib.bh_compute_forces.argtypes = [C.c_void_p, C.c_float, C.c_float, C.c_void_p]
    lib.bh_refresh_moments.argtypes = [C.c_void_p, C.c_void_p]
    lib.bh_refresh_moments.restype = C.c_int
    lib.bh_compute_forces_active.argtypes = [C.c_void_p, C.c_float, C.c_float, C.c_void_p, C.c_void_p]
    lib.bh_compute_forces_active.restype = C.c_int
    lib.bh_refresh_moments_active.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
    lib.bh_refresh_moments_active.restype = C.c_int
    lib.bh_block_init.argtypes = [C.c_void_p, C.POINTER(BhBlockConfig), C.c_void_p]
    lib.bh_block_init.restype = C.c_int
    lib.bh_block_step.argtypes = [C.c_void_p, C.c_float, C.c_float, C.c_int, C.c_void_p]
    lib.bh_block_step.restype = C.c_int
    lib.bh_block_state.argtypes = [C.c_void_p, C.POINTER(BhBlockStats), C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    lib.bh_block_state.restype = C.c_int
    lib.bh_set_mac.argtypes = [C.c_void_p, C.c_int]
    lib.bh_set_mac.restype = C.c_int
    lib.bh_leapfrog_step.argtypes = [C.c_void_p, C.c_float, C.c_float, C.c_float, C.c_void_p]
    lib.bh_kick_drift.argtypes = [C.c_void_p, C.c_float, C.c_float, C.c_void_p]
    lib.bh_step_graph_build.argtypes = [C.c_void_p, C.c_float, C.c_float, C.c_float, C.c_void_p]
    lib.bh_step_graph_build.restype = C.c_int
    lib.bh_step_graph_launch.argtypes = [C.c_void_p, C.c_void_p]
    lib.bh_step_graph_launch.restype = C.c_int
    lib.bh_sync_status.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(BhStats)]
    lib.bh_export_tree.argtypes = [C.c_void_p, C.POINTER(BhTreeView), C.c_void_p]
    lib.bh_set_stage_timing.argtypes = [C.c_void_p, C.c_int]
    lib.bh_get_stage_ms.argtypes = [C.c_void_p, C.POINTER(C.c_float)]
    lib.bh_get_walk_timeline.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(C.c_int64), C.c_int]
    lib.bh_get_walk_timeline.restype = C.c_int
    lib.bh_direct_forces.argtypes = [C.c_void_p, C.c_int64, C.c_float, C.c_int64, C.c_int64, C.c_void_p, C.c_void_p]
    lib.bh_direct_forces.restype = C.c_int
    lib.bh_domain_box_static.argtypes = [C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p]
    lib.bh_domain_box_static.restype = C.c_int
    lib.bh_domain_box_static_max_n.argtypes = []
    lib.bh_domain_box_static_max_n.restype = C.c_int64
    lib.bh_probe_fp32.argtypes = [C.c_int, C.c_void_p, C.c_size_t, C.POINTER(C.c_double), C.POINTER(C.c_double)]
    lib.bh_probe_fp32.restype = C.c_int
    lib.bh_last_cuda_error.argtypes = [C.c_void_p]
    lib.bh_status_string.restype = C.c_char_p
    lib.bh_status_string.argtypes = [C.c_int]
    for f in ("bh_create", "bh_destroy", "bh_set_particles", "bh_get_particles", "bh_tree_build", "bh_compute_forces",
              "bh_leapfrog_step", "bh_kick_drift", "bh_sync_status", "bh_export_tree", "bh_set_stage_timing", "bh_get_stage_ms",
              "bh_last_cuda_error"):
        getattr(lib, f).restype = C.c_int
    _lib = lib
    return lib


def workspace_bytes(n_max: int, nleaf: int = 0, ncrit: int = 0, max_cells: int = 0, list_entries: int = 0, walk_mode: int = 0,
                    walk_waves: int = 0, front_mode: int = 0, walk_private: int = 0) -> int:
    cfg = BhConfig(nleaf, ncrit, max_cells, list_entries, walk_mode, walk_waves, front_mode, walk_private)
    return int(load_library().bh_workspace_bytes(n_max, C.byref(cfg)))


def direct_forces(pos_mass: torch.Tensor, eps: float, t0: int = 0, t1: int | None = None, out: torch.Tensor | None = None) -> torch.Tensor:
    """bh_direct_forces: binary64 O(N^2) direct sum on the GPU for targets [t0, t1).  pos_mass: CUDA float32[n,4];
    returns (or fills) a CUDA float64[n,4] tensor (ax, ay, az, phi); rows outside the range are left as they are (NaN if new)."""
    if not (pos_mass.is_cuda and pos_mass.dtype == torch.float32 and pos_mass.is_contiguous() and pos_mass.dim() == 2 and pos_mass.shape[1] == 4):
        raise BhError(-1, "pos_mass must be a contiguous CUDA float32[n,4] tensor")
    n = int(pos_mass.shape[0])
    t1 = n if t1 is None else t1
    if out is None:
        out = torch.full((n, 4), float("nan"), dtype=torch.float64, device=pos_mass.device)
    assert out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and tuple(out.shape) == (n, 4)
    rc = load_library().bh_direct_forces(pos_mass.data_ptr(), n, eps, t0, t1, out.data_ptr(),
                                         C.c_void_p(torch.cuda.current_stream(pos_mass.device).cuda_stream))
    if rc != BH_OK:
        raise BhError(rc, "bh_direct_forces")
    return out


def domain_box_static_max_n() -> int:
    """Most particles bh_domain_box_static accepts (the size of its built-in scratch array fixes it)."""
    return int(load_library().bh_domain_box_static_max_n())


def domain_box_static(pos_mass: torch.Tensor, out: torch.Tensor) -> torch.Tensor:
    """bh_domain_box_static: the S0 domain box of ``pos_mass`` (CUDA float32[n,4]) without a context, a workspace or any
    allocation by the library -- for callers that have no device memory to hand over and may not call cudaMalloc (all of the
    card owned by another allocator, a fixed memory budget, a loop that cannot take cudaMalloc's device-wide stall).

    ``out``: a CUDA int32[8] tensor on the same device that the CALLER provides (this wrapper allocates nothing either); the
    kernel fills it with the 32 bytes of ``bh_domain_box``: lo xyz and hi xyz as float32 bit patterns, domain_exp, status.
    Only enqueues work on the current stream of that device and returns ``out``; decode it with ``decode_domain_box`` after
    synchronising.  n above ``domain_box_static_max_n()`` raises BhError(BH_ERR_TOO_LARGE).  All calls on one GPU share one
    scratch array inside the library: keep them on one stream (or otherwise ordered); overlapping calls race.  The first call
    on a device also looks up that array's address, so make it during set-up."""
    if not (pos_mass.is_cuda and pos_mass.dtype == torch.float32 and pos_mass.is_contiguous() and pos_mass.dim() == 2 and pos_mass.shape[1] == 4):
        raise BhError(-1, "pos_mass must be a contiguous CUDA float32[n,4] tensor")
    if not (out.is_cuda and out.dtype == torch.int32 and out.is_contiguous() and out.numel() == 8 and out.device == pos_mass.device):
        raise BhError(-1, "out must be a contiguous CUDA int32[8] tensor on the device of pos_mass")
    n = int(pos_mass.shape[0])
    rc = load_library().bh_domain_box_static(pos_mass.data_ptr(), n, out.data_ptr(),
                                             C.c_void_p(torch.cuda.current_stream(pos_mass.device).cuda_stream))
    if rc != BH_OK:
        what = f"bh_domain_box_static: n = {n} exceeds the limit of {domain_box_static_max_n()} particles" if rc == -7 else "bh_domain_box_static"
        raise BhError(rc, what)
    return out


def decode_domain_box(out: torch.Tensor) -> BhDomainBox:
    """The int32[8] result of ``domain_box_static`` as a BhDomainBox (copies 32 bytes to the host: synchronises)."""
    raw = out.detach().cpu().numpy().astype(np.int32, copy=False).tobytes()
    return BhDomainBox.from_buffer_copy(raw)


PROBE_KINDS = {"ffma": 0, "ffma2": 1, "ffma2_shared_operand": 2, "ffma2_broadcast_scalar": 3, "pc_body": 4, "pp_body": 5}


def probe_fp32(device=None) -> dict:
    """bh_probe_fp32 for every kind: {name: TFLOP/s} (+ "<body>_executed" for the force bodies).  Synchronises."""
    lib = load_library()
    dev = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
    sms = torch.cuda.get_device_properties(dev).multi_processor_count
    scratch = torch.empty(sms * 512 + 4096, dtype=torch.float32, device=dev)
    torch.cuda.synchronize(dev)
    out = {}
    with torch.cuda.device(dev):
        for name, kind in PROBE_KINDS.items():
            a, b = C.c_double(0.0), C.c_double(0.0)
            rc = lib.bh_probe_fp32(kind, scratch.data_ptr(), scratch.numel() * 4, C.byref(a), C.byref(b))
            if rc != BH_OK:
                raise BhError(rc, "bh_probe_fp32")
            out[name] = a.value
            if kind >= 4:
                out[name + "_executed"] = b.value
    return out


STAGES = ["bbox", "keys", "sort", "reorder", "cells", "groups", "moments", "record", "walk", "lists", "eval"]


def _ptr(x):
    """Host (numpy / pinned torch) or device (torch cuda) buffer -> raw pointer; None -> NULL."""
    if x is None:
        return None
    if isinstance(x, np.ndarray):
        assert x.flags["C_CONTIGUOUS"]
        return x.ctypes.data
    assert x.is_contiguous()
    return x.data_ptr()


class BarnesHut:
    """One Barnes-Hut context on one GPU: same calls as include/bh.h (bh_tree_build, bh_compute_forces, bh_leapfrog_step)."""

    def __init__(self, n_max: int, nleaf: int = 0, ncrit: int = 0, max_cells: int = 0, list_entries: int = 0, walk_mode: int = 0,
                 walk_waves: int = 0, front_mode: int = 0, walk_private: int = 0, device=None):
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1106_1900_b200 needs a CUDA device: there is no CPU fallback")
        self.lib = load_library()
        self.device = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
        cfg = BhConfig(nleaf, ncrit, max_cells, list_entries, walk_mode, walk_waves, front_mode, walk_private)
        nbytes = int(self.lib.bh_workspace_bytes(n_max, C.byref(cfg)))
        if nbytes == 0:
            raise BhError(-1, "bad n_max / config")
        self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        base = (self.workspace.data_ptr() + 255) & ~255
        self._ws_off = base - self.workspace.data_ptr()
        self._ws_base = base
        self._ws_bytes = nbytes
        h = C.c_void_p()
        self._check(self.lib.bh_create(C.byref(h), n_max, C.byref(cfg), C.c_void_p(base), nbytes), "bh_create")
        self.h = h
        self.n_max = n_max
        self.n = 0

    # ------------------------------------------------------------------ helpers
    def _check(self, rc: int, what: str = ""):
        if rc != BH_OK:
            extra = ""
            if rc == -4 and getattr(self, "h", None):
                extra = f" (cudaError {self.lib.bh_last_cuda_error(self.h)})"
            raise BhError(rc, what + extra)

    def _stream(self):
        return C.c_void_p(torch.cuda.current_stream(self.device).cuda_stream)

    def close(self):
        if getattr(self, "h", None):
            self.lib.bh_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ------------------------------------------------------------------ the C ABI, one to one
    def set_particles(self, pos_mass, vel=None, ids=None):
        """pos_mass float32[n,4], vel float32[n,4] or None, ids uint32[n] or None; numpy, pinned or CUDA torch tensors."""
        n = int(pos_mass.shape[0])
        self._keep = (pos_mass, vel, ids)   # keep host buffers alive until the async copies are done
        self._check(self.lib.bh_set_particles(self.h, n, _ptr(pos_mass), _ptr(vel), _ptr(ids), self._stream()), "bh_set_particles")
        if getattr(self, "_bound", None) is not None:
            self._bound = None             # back to the workspace's own arrays
            self._acc_ptr = None
        self.n = n

    def bind_particles(self, pos_mass: torch.Tensor, vel: torch.Tensor, acc_pot: torch.Tensor, ids: torch.Tensor):
        """bh_bind_particles: the caller's CUDA tensors (float32[n,4] x 3, int32[n] ids) become the simulation state; no copy.
        The tensors are kept alive by this object until set_particles / another bind_particles / close."""
        n = int(pos_mass.shape[0])
        for t, shape, dt in ((pos_mass, (n, 4), torch.float32), (vel, (n, 4), torch.float32), (acc_pot, (n, 4), torch.float32), (ids, (n,), torch.int32)):
            if not (t.is_cuda and t.device == self.device and t.dtype == dt and t.is_contiguous() and tuple(t.shape) == shape):
                raise BhError(-1, "bind_particles wants contiguous CUDA tensors on this device: float32[n,4] x 3 and int32[n]")
        self._check(self.lib.bh_bind_particles(self.h, n, pos_mass.data_ptr(), vel.data_ptr(), acc_pot.data_ptr(), ids.data_ptr()), "bh_bind_particles")
        self._bound = (pos_mass, vel, acc_pot, ids)
        self._acc_ptr = None
        self.n = n

    def land_particles(self):
        """bh_land_particles: make the bound tensors hold the current sorted state (one device copy, or nothing)."""
        self._check(self.lib.bh_land_particles(self.h, self._stream()), "bh_land_particles")

    def get_particles(self, pos_mass=None, vel=None, acc_pot=None, ids=None):
        self._check(self.lib.bh_get_particles(self.h, _ptr(pos_mass), _ptr(vel), _ptr(acc_pot), _ptr(ids), self._stream()),
                    "bh_get_particles")

    def tree_build(self):
        self._check(self.lib.bh_tree_build(self.h, self._stream()), "bh_tree_build")

    def compute_forces(self, theta: float, eps: float):
        self._check(self.lib.bh_compute_forces(self.h, theta, eps, self._stream()), "bh_compute_forces")

    def refresh_moments(self):
        """S6 on the existing cells after the particles moved (block time-steps)."""
        self._check(self.lib.bh_refresh_moments(self.h, self._stream()), "bh_refresh_moments")

    def compute_forces_active(self, theta: float, eps: float, active: torch.Tensor):
        """S7 + S8 for the groups with an active particle; active: CUDA uint8[n] in the current sorted order."""
        if not (active.is_cuda and active.dtype == torch.uint8 and active.is_contiguous() and active.numel() == self.n):
            raise BhError(-1, "active must be a contiguous CUDA uint8[n] tensor")
        self._keep_active = active
        self._check(self.lib.bh_compute_forces_active(self.h, theta, eps, active.data_ptr(), self._stream()), "bh_compute_forces_active")

    def refresh_moments_active(self, active: torch.Tensor):
        """S6 only for the cells above an active particle; active: CUDA uint8[n] in the current sorted order."""
        if not (active.is_cuda and active.dtype == torch.uint8 and active.is_contiguous() and active.numel() == self.n):
            raise BhError(-1, "active must be a contiguous CUDA uint8[n] tensor")
        self._keep_active = active
        self._check(self.lib.bh_refresh_moments_active(self.h, active.data_ptr(), self._stream()), "bh_refresh_moments_active")

    def block_init(self, len_scale: float, eta: float, dt_max: float, max_rung: int):
        """Block time-steps (include/bh.h): all particles at tick 0 with the current forces, rungs from the criterion."""
        cfg = BhBlockConfig(len_scale, eta, dt_max, max_rung)
        self._check(self.lib.bh_block_init(self.h, C.byref(cfg), self._stream()), "bh_block_init")

    def block_step(self, theta: float, eps: float, rebuild: bool = False):
        """One system step of the block scheme: active set, predictor, moments (or rebuild), walk of the active groups, corrector."""
        self._check(self.lib.bh_block_step(self.h, theta, eps, int(bool(rebuild)), self._stream()), "bh_block_step")

    def block_state(self, arrays: bool = True) -> dict:
        """bh_block_state: stats (+ tick uint32[n], rung uint8[n], active uint8[n], acc_held float32[n,4] as numpy); synchronises."""
        st = BhBlockStats()
        out = {}
        if arrays:
            n = self.n
            out = dict(tick=np.empty(n, np.uint32), rung=np.empty(n, np.uint8), active=np.empty(n, np.uint8), acc_held=np.empty((n, 4), np.float32))
            self._check(self.lib.bh_block_state(self.h, C.byref(st), _ptr(out["tick"]), _ptr(out["rung"]), _ptr(out["active"]),
                                                _ptr(out["acc_held"]), self._stream()), "bh_block_state")
        else:
            self._check(self.lib.bh_block_state(self.h, C.byref(st), None, None, None, None, self._stream()), "bh_block_state")
        out["stats"] = st
        return out

    def set_mac(self, mac: int):
        """0: Eq.1 (default); 1: minimum-distance MAC."""
        self._check(self.lib.bh_set_mac(self.h, int(mac)), "bh_set_mac")

    def leapfrog_step(self, theta: float, eps: float, dt: float):
        self._check(self.lib.bh_leapfrog_step(self.h, theta, eps, dt, self._stream()), "bh_leapfrog_step")

    def step_graph_build(self, theta: float, eps: float, dt: float):
        """Capture bh_leapfrog_step(theta, eps, dt) into CUDA graphs owned by the context (nothing runs)."""
        self._check(self.lib.bh_step_graph_build(self.h, theta, eps, dt, self._stream()), "bh_step_graph_build")

    def step_graph_launch(self):
        """One captured step: bh_leapfrog_step as a single graph launch."""
        self._check(self.lib.bh_step_graph_launch(self.h, self._stream()), "bh_step_graph_launch")

    def kick_drift(self, dt_kick: float, dt_drift: float):
        self._check(self.lib.bh_kick_drift(self.h, dt_kick, dt_drift, self._stream()), "bh_kick_drift")

    def sync_status(self, check: bool = True) -> BhStats:
        st = BhStats()
        rc = self.lib.bh_sync_status(self.h, self._stream(), C.byref(st))
        if check:
            self._check(rc, "bh_sync_status")
        return st

    def set_stage_timing(self, enable: bool):
        self._check(self.lib.bh_set_stage_timing(self.h, int(enable)))

    def stage_ms(self) -> dict:
        ms = (C.c_float * 11)()
        self._check(self.lib.bh_get_stage_ms(self.h, ms), "bh_get_stage_ms")
        return dict(zip(STAGES, [float(x) for x in ms]))

    def walk_timeline(self, max_waves: int = 256):
        """[(lists_start, lists_end, eval_start, eval_end)] per wave of the last walk, ns relative to the first start."""
        buf = (C.c_int64 * (4 * max_waves))()
        w = self.lib.bh_get_walk_timeline(self.h, self._stream(), buf, max_waves)
        if w < 0:
            self._check(w, "bh_get_walk_timeline")
        t0 = min(buf[4 * i] for i in range(w)) if w else 0
        return [tuple(int(buf[4 * i + j] - t0) for j in range(4)) for i in range(w)]

    # ------------------------------------------------------------------ views of the workspace (no copies)
    def _view(self, ptr: int, count: int, dtype: torch.dtype, shape=None):
        if ptr is None or count == 0:
            return torch.empty(0, dtype=dtype, device=self.device)
        for t in (getattr(self, "_bound", None) or ()):          # bh_bind_particles: the pointer may be one of the caller's tensors
            if t.data_ptr() == ptr:
                return t.view(dtype).view(shape) if shape is not None else t.view(dtype).reshape(-1)
        off = ptr - self.workspace.data_ptr()
        nb = count * torch.empty(0, dtype=dtype).element_size()
        t = self.workspace[off: off + nb].view(dtype)
        return t.view(shape) if shape is not None else t

    def acc_view(self) -> torch.Tensor:
        """float32[n,4] view of the acc_pot array in the workspace (no copy, no synchronisation)."""
        v = BhTreeView()
        # bh_export_tree would enqueue the export kernel; the acc array sits at a fixed place of the workspace, so ask once
        if getattr(self, "_acc_ptr", None) is None:
            self._check(self.lib.bh_export_tree(self.h, C.byref(v), self._stream()), "bh_export_tree")
            self._acc_ptr = v.acc_pot
        return self._view(self._acc_ptr, self.n * 4, torch.float32, (self.n, 4))

    def group_views(self):
        """(group_begin int32[G+1], group_npc int32[G], group_npp int32[G]) as views of the workspace; synchronises (the group
        count lives on the device).  No export kernel is launched."""
        if getattr(self, "_group_ptrs", None) is None:
            v = BhTreeView()
            self._check(self.lib.bh_export_tree(self.h, C.byref(v), self._stream()), "bh_export_tree")
            self._group_ptrs = (v.group_begin, v.group_npc, v.group_npp)
        ng = int(self.sync_status().n_groups)
        pb, pc, pp = self._group_ptrs
        i32 = torch.int32
        return self._view(pb, ng + 1, i32), self._view(pc, ng, i32), self._view(pp, ng, i32)

    def export_tree(self) -> dict:
        """Canonical arrays of bh_tree_view as torch tensors that alias the workspace (synchronises)."""
        v = BhTreeView()
        self._check(self.lib.bh_export_tree(self.h, C.byref(v), self._stream()), "bh_export_tree")
        st = self.sync_status()
        n, nc, ng = int(st.n), int(st.n_cells), int(st.n_groups)
        f32, i32, u8 = torch.float32, torch.int32, torch.uint8
        out = dict(stats=st, n=n, n_cells=nc, n_groups=ng)
        out["pos_mass"] = self._view(v.pos_mass, n * 4, f32, (n, 4))
        out["vel"] = self._view(v.vel, n * 4, f32, (n, 4))
        out["acc_pot"] = self._view(v.acc_pot, n * 4, f32, (n, 4))
        out["id"] = self._view(v.id, n, i32)                 # uint32 payload viewed as int32 (n < 2^31)
        out["key"] = self._view(v.key, n, torch.int64)       # 60-bit keys fit a signed 64-bit view
        out["perm"] = self._view(v.perm, n, i32)
        out["level_offset"] = self._view(v.level_offset, 22, i32)
        out["cell_level"] = self._view(v.cell_level, nc, i32)
        out["cell_prefix"] = self._view(v.cell_prefix, nc, torch.int64)
        out["cell_pbegin"] = self._view(v.cell_pbegin, nc, i32)
        out["cell_pcount"] = self._view(v.cell_pcount, nc, i32)
        out["cell_child_begin"] = self._view(v.cell_child_begin, nc, i32)
        out["cell_nchild"] = self._view(v.cell_nchild, nc, i32)
        out["cell_parent"] = self._view(v.cell_parent, nc, i32)
        out["cell_mom64"] = self._view(v.cell_mom64, nc * 10, torch.float64, (nc, 10))
        out["cell_box"] = self._view(v.cell_box, nc * 6, f32, (nc, 6))
        out["cell_mom32"] = self._view(v.cell_mom32, nc * 10, f32, (nc, 10))
        out["cell_r2open"] = self._view(v.cell_r2open, nc, f32)
        out["cell_trec"] = self._view(v.cell_trec, nc * 4, f32, (nc, 4))
        out["cell_erec"] = self._view(v.cell_erec, nc * 12, f32, (nc, 12))
        out["group_begin"] = self._view(v.group_begin, ng + 1, i32)
        out["group_cell"] = self._view(v.group_cell, ng, i32)
        out["group_npc"] = self._view(v.group_npc, ng, i32)
        out["group_npp"] = self._view(v.group_npp, ng, i32)
        return out
