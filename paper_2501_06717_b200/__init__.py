"""Thin Python binding of the C-ABI library declared in include/batl.h.

Argument marshalling only: every step of the hot path (ghost fill, face
reconstruction, Rusanov flux, sources, update, dt reduction) runs in the CUDA
kernels of ``csrc/``.  PyTorch is used for device memory and the CUDA stream,
nothing else.  There is no CPU fallback: binding a grid without the compiled
library or without a CUDA device raises.

The function names mirror the C entry points (batl_init_grid, batl_bind,
batl_set_state, mhd_step, batl_get_state, ...); ``Grid`` bundles them with the
torch-owned buffers for convenience.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import _build

NI, NG, NS, NV = 8, 2, 12, 8
BLOCK_BYTES = NV * NS ** 3 * 8

BC_PERIODIC, BC_FLOAT, BC_FIXED = 0, 1, 2
SHAPE_ALL, SHAPE_BOX, SHAPE_SPHERE = 0, 1, 2
DT_GLOBAL, DT_LOCAL, DT_FIXED = 0, 1, 2
LIST_MESSAGES, LIST_EXPANDED, LIST_PLAN, LIST_PLAN_PATTERNS = 0, 1, 2, 3
WARN_NONFINITE, WARN_NEGATIVE = 1, 2

EXPORTS = (
    "batl_init_grid", "batl_free_grid", "batl_n_blocks", "batl_buffer_bytes", "batl_bind",
    "batl_set_state", "batl_set_state_device", "mhd_step", "mhd_step_async", "batl_fill_ghosts",
    "batl_get_state", "batl_get_dt_local", "batl_get_blocks", "batl_get_neighbors",
    "batl_get_ghost_list", "batl_set_kernel_variant", "batl_phase_timers", "batl_launch_count",
    "batl_kernel_counts", "batl_last_error",
    "batl_set_partition", "batl_get_partition", "batl_bind_peers", "batl_step_part", "batl_scalar_offsets",
    "mhd_stable_dt_static", "batl_static_last_error",
)


class BatlRegion(C.Structure):
    _fields_ = [("shape", C.c_int32), ("level", C.c_int32), ("p", C.c_double * 6)]


class BatlConfig(C.Structure):
    _fields_ = [
        ("n_root", C.c_int32 * 3),
        ("xyz_min", C.c_double * 3), ("xyz_max", C.c_double * 3),
        ("bc", C.c_int32 * 6),
        ("bc_prim", (C.c_double * 8) * 6),
        ("n_region", C.c_int32),
        ("region", C.POINTER(BatlRegion)),
        ("max_level", C.c_int32),
        ("gamma", C.c_double), ("cfl", C.c_double), ("limiter_beta", C.c_double),
        ("dt_mode", C.c_int32), ("dt_fixed", C.c_double),
        ("use_divb_source", C.c_int32),
        ("use_b0", C.c_int32), ("dipole_m", C.c_double * 3),
        ("use_body", C.c_int32),
        ("r_body", C.c_double), ("rho_body", C.c_double), ("p_body", C.c_double),
        ("n_stage", C.c_int32), ("n_order", C.c_int32), ("flux_type", C.c_int32),
        ("prolong_order", C.c_int32), ("flux_correction", C.c_int32),
    ]


GHOST_MSG_DTYPE = np.dtype([("dst", "<i4"), ("src", "<i4"), ("kind", "i1"), ("dir", "i1"),
                            ("lo", "i1", 3), ("n", "i1", 3), ("mul", "i1", 3), ("off", "i1", 3),
                            ("shift", "i1", 3), ("pad", "i1", 3)])
assert GHOST_MSG_DTYPE.itemsize == 28

_lib = None


class BatlError(RuntimeError):
    pass


def lib():
    """Loads (building it first if the sources are newer) the C-ABI library."""
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        vp, sp = C.c_void_p, C.POINTER(C.c_size_t)
        L.batl_init_grid.argtypes = [C.POINTER(BatlConfig), C.POINTER(vp)]
        L.batl_free_grid.argtypes = [vp]
        L.batl_free_grid.restype = None
        L.batl_n_blocks.argtypes = [vp, C.POINTER(C.c_int32)]
        L.batl_buffer_bytes.argtypes = [vp, sp, sp]
        L.batl_bind.argtypes = [vp, vp, vp, vp, vp]
        L.batl_set_state.argtypes = [vp, vp]
        L.batl_set_state_device.argtypes = [vp, vp]
        L.mhd_step.argtypes = [vp, C.c_int32, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.mhd_step_async.argtypes = [vp, C.c_int32]
        L.batl_fill_ghosts.argtypes = [vp]
        L.batl_get_state.argtypes = [vp, vp, C.c_int32]
        L.batl_get_dt_local.argtypes = [vp, vp]
        L.batl_get_blocks.argtypes = [vp, vp]
        L.batl_get_neighbors.argtypes = [vp, vp, vp]
        L.batl_get_ghost_list.argtypes = [vp, C.c_int32, vp, sp]
        L.batl_set_kernel_variant.argtypes = [vp, C.c_int32]
        L.batl_phase_timers.argtypes = [vp, C.c_int32] + [C.POINTER(C.c_double)] * 3
        L.batl_launch_count.argtypes = [vp, C.POINTER(C.c_int64)]
        L.batl_kernel_counts.argtypes = [vp, C.POINTER(C.c_int64)]
        L.batl_set_partition.argtypes = [vp, C.c_int32, C.c_int32]
        L.batl_get_partition.argtypes = [vp, vp]
        L.batl_bind_peers.argtypes = [vp, vp, vp]
        L.batl_step_part.argtypes = [vp, C.c_int32]
        L.batl_scalar_offsets.argtypes = [vp, sp]
        L.batl_last_error.restype = C.c_char_p
        L.mhd_stable_dt_static.argtypes = [vp, vp, C.c_int32, C.c_double, C.c_double, C.c_double, C.c_int32, C.c_int32,
                                           C.c_int32, vp, vp, vp]
        L.batl_static_last_error.restype = C.c_char_p
        _lib = L
    return _lib


def _check(rc):
    if rc < 0:
        raise BatlError(f"batl error {rc}: {lib().batl_last_error().decode()}")
    return rc


def make_config(cfg: dict):
    """dict (the layout of workloads/*.py) -> (BatlConfig, keep-alive objects)."""
    c = BatlConfig()
    for a in range(3):
        c.n_root[a] = int(cfg["n_root"][a])
        c.xyz_min[a] = float(cfg["xyz_min"][a])
        c.xyz_max[a] = float(cfg["xyz_max"][a])
        c.dipole_m[a] = float(cfg["dipole_m"][a])
    bp = np.asarray(cfg["bc_prim"], dtype=np.float64).reshape(6, 8)
    for f in range(6):
        c.bc[f] = int(cfg["bc"][f])
        for v in range(8):
            c.bc_prim[f][v] = float(bp[f, v])
    regs = cfg["regions"]
    arr = (BatlRegion * max(1, len(regs)))()
    for r, (shape, level, p) in enumerate(regs):
        arr[r].shape, arr[r].level = int(shape), int(level)
        for q in range(6):
            arr[r].p[q] = float(p[q])
    c.n_region = len(regs)
    c.region = C.cast(arr, C.POINTER(BatlRegion))
    c.max_level = int(cfg["max_level"])
    c.gamma, c.cfl, c.limiter_beta = float(cfg["gamma"]), float(cfg["cfl"]), float(cfg["limiter_beta"])
    c.dt_mode, c.dt_fixed = int(cfg["dt_mode"]), float(cfg["dt_fixed"])
    c.use_divb_source = int(cfg["use_divb_source"])
    c.use_b0 = int(cfg["use_b0"])
    c.use_body = int(cfg["use_body"])
    c.r_body, c.rho_body, c.p_body = float(cfg["r_body"]), float(cfg["rho_body"]), float(cfg["p_body"])
    c.n_stage, c.n_order = int(cfg.get("n_stage", 2)), int(cfg.get("n_order", 2))
    c.flux_type = int(cfg.get("flux_type", 0))
    c.prolong_order = int(cfg.get("prolong_order", 1))
    c.flux_correction = int(cfg.get("flux_correction", 0))
    return c, arr


class Grid:
    """One batl_grid.  The host part (tree, tables, ghost lists) needs no GPU;
    ``bind()`` allocates the device buffers with torch and attaches them."""

    def __init__(self, cfg: dict):
        L = lib()
        self.cfg = cfg
        c, keep = make_config(cfg)
        h = C.c_void_p()
        _check(L.batl_init_grid(C.byref(c), C.byref(h)))
        self._h = h
        n = C.c_int32()
        _check(L.batl_n_blocks(self._h, C.byref(n)))
        self.n_blocks = n.value
        sb, wb = C.c_size_t(), C.c_size_t()
        _check(L.batl_buffer_bytes(self._h, C.byref(sb), C.byref(wb)))
        self.state_bytes, self.scratch_bytes = sb.value, wb.value
        self._bufs = None
        self.stream = None
        self.world, self.rank = 1, 0

    def close(self):
        if getattr(self, "_h", None):
            if _lib is not None:             # None once the interpreter is tearing the module down
                _lib.batl_free_grid(self._h)
            self._h = None
        self._bufs = None

    def __del__(self):
        self.close()

    # ---- host introspection (no GPU) -----------------------------------------
    def blocks(self):
        out = np.zeros((self.n_blocks, 4), dtype=np.int32)
        _check(lib().batl_get_blocks(self._h, out.ctypes.data))
        return out

    def neighbors(self):
        nbr = np.zeros((self.n_blocks, 27, 4), dtype=np.int32)
        dlev = np.zeros((self.n_blocks, 27), dtype=np.int8)
        _check(lib().batl_get_neighbors(self._h, nbr.ctypes.data, dlev.ctypes.data))
        return nbr, dlev

    def ghost_list(self, from_plan=False):
        """Canonical per-ghost-cell tuples, expanded from the message records or (from_plan)
        decoded from the per-cell plan the ghost-fill kernel reads."""
        kind = LIST_PLAN if from_plan else LIST_EXPANDED
        n = C.c_size_t()
        _check(lib().batl_get_ghost_list(self._h, kind, None, C.byref(n)))
        out = np.zeros((n.value, 9), dtype=np.int32)
        _check(lib().batl_get_ghost_list(self._h, kind, out.ctypes.data, C.byref(n)))
        return out

    def plan_patterns(self):
        n = C.c_size_t()
        _check(lib().batl_get_ghost_list(self._h, LIST_PLAN_PATTERNS, None, C.byref(n)))
        out = np.zeros((n.value, 1216), dtype=np.uint32)
        _check(lib().batl_get_ghost_list(self._h, LIST_PLAN_PATTERNS, out.ctypes.data, C.byref(n)))
        return out

    def _int_list(self, kind, width):
        n = C.c_size_t()
        _check(lib().batl_get_ghost_list(self._h, kind, None, C.byref(n)))
        out = np.zeros((n.value, width) if width > 1 else (n.value,), dtype=np.int32)
        if n.value:
            _check(lib().batl_get_ghost_list(self._h, kind, out.ctypes.data, C.byref(n)))
        return out

    def plan_ids(self):
        """Pattern (row of plan_patterns()) of every block."""
        return self._int_list(4, 1)

    def flux_correction_tables(self):
        """(slots[nB][6], records[n][8]) of batl.h BATL_LIST_FC_SLOTS / BATL_LIST_FC_RECORDS."""
        return self._int_list(5, 6), self._int_list(6, 8)

    def ghost_messages(self):
        n = C.c_size_t()
        _check(lib().batl_get_ghost_list(self._h, LIST_MESSAGES, None, C.byref(n)))
        out = np.zeros(n.value, dtype=GHOST_MSG_DTYPE)
        _check(lib().batl_get_ghost_list(self._h, LIST_MESSAGES, out.ctypes.data, C.byref(n)))
        return out

    # ---- device side ---------------------------------------------------------
    def bind(self, device="cuda:0", stream=None):
        import torch
        if not torch.cuda.is_available():
            raise BatlError("no CUDA device: the MHD step has no CPU path")
        dev = torch.device(device)
        torch.cuda.set_device(dev)
        self.stream = stream if stream is not None else torch.cuda.current_stream(dev)
        with torch.cuda.stream(self.stream):
            A = torch.zeros(max(1, self.state_bytes // 8), dtype=torch.float64, device=dev)
            B = torch.zeros(max(1, self.state_bytes // 8), dtype=torch.float64, device=dev)
            S = torch.zeros(max(256, self.scratch_bytes), dtype=torch.uint8, device=dev)
        self._bufs = (A, B, S)
        _check(lib().batl_bind(self._h, A.data_ptr(), B.data_ptr(), S.data_ptr(), self.stream.cuda_stream))
        return self

    def set_state(self, U):
        """U: host array [nB][8][8][8][8] (conserved) or a CUDA float64 tensor of that shape."""
        try:
            import torch
            is_tensor = isinstance(U, torch.Tensor)
        except ImportError:      # pragma: no cover
            is_tensor = False
        if is_tensor and U.is_cuda:
            assert U.dtype == torch.float64 and U.is_contiguous() and U.numel() == self.n_blocks * NV * NI ** 3
            # batl.h: the copy is enqueued on the bound stream, which knows nothing of the stream that
            # produced U -- order the two here, and keep U's memory from being reused before the copy ran
            self.stream.wait_stream(torch.cuda.current_stream(U.device))
            U.record_stream(self.stream)
            _check(lib().batl_set_state_device(self._h, U.data_ptr()))
            return
        if is_tensor:
            assert U.dtype == torch.float64 and U.is_contiguous() and U.numel() == self.n_blocks * NV * NI ** 3
            _check(lib().batl_set_state(self._h, U.data_ptr()))
            return
        U = np.ascontiguousarray(U, dtype=np.float64)
        assert U.shape == (self.n_blocks, NV, NI, NI, NI)
        _check(lib().batl_set_state(self._h, U.ctypes.data))

    def step(self, n_steps=1):
        """Returns (warning bitmask, t, dt_last); waits for the stream."""
        t, dt = C.c_double(0.0), C.c_double(0.0)
        w = _check(lib().mhd_step(self._h, int(n_steps), C.byref(t), C.byref(dt)))
        return w, t.value, dt.value

    def step_async(self, n_steps=1):
        _check(lib().mhd_step_async(self._h, int(n_steps)))

    def fill_ghosts(self):
        _check(lib().batl_fill_ghosts(self._h))

    def get_state(self, with_ghost=False, out=None):
        """with_ghost: False / True, or 2 = the stored 12^3 tiles as they are (batl.h)."""
        n = NS if with_ghost else NI
        if out is None:
            out = np.zeros((self.n_blocks, NV, n, n, n))
            _check(lib().batl_get_state(self._h, out.ctypes.data, int(with_ghost)))
            return out
        _check(lib().batl_get_state(self._h, out.data_ptr(), int(with_ghost)))   # pinned torch tensor
        return out

    def get_dt_local(self):
        out = np.zeros((self.n_blocks, NI, NI, NI))
        _check(lib().batl_get_dt_local(self._h, out.ctypes.data))
        return out

    def set_kernel_variant(self, variant: int):
        _check(lib().batl_set_kernel_variant(self._h, int(variant)))

    def phase_timers(self, enable: bool):
        a, b, c = C.c_double(), C.c_double(), C.c_double()
        _check(lib().batl_phase_timers(self._h, int(enable), C.byref(a), C.byref(b), C.byref(c)))
        return dict(stage_ms=a.value, ghost_ms=b.value, other_ms=c.value)

    def kernel_counts(self):
        """dict of batl_kernel_counts: which kernels mhd_step used (general_fallback > 0 means the
        fused kernel had no instantiation for this configuration)."""
        out = (C.c_int64 * 6)()
        _check(lib().batl_kernel_counts(self._h, out))
        keys = ("fused", "general", "general_fallback", "fill_launches", "fill_blocks", "fill_list")
        return dict(zip(keys, (int(x) for x in out)))

    # ---- sharding over the GPUs of one node (batl.h) -----------------------------
    def set_partition(self, world: int, rank: int):
        """Before bind(): this process owns the rank-th contiguous Morton segment of the blocks."""
        _check(lib().batl_set_partition(self._h, int(world), int(rank)))
        self.world, self.rank = int(world), int(rank)
        return self

    def partition(self):
        out = np.zeros(self.world + 1, dtype=np.int32)
        _check(lib().batl_get_partition(self._h, out.ctypes.data))
        return out

    def bind_peers(self, ptrs_A, ptrs_B):
        """ptrs_A / ptrs_B: device addresses of every rank's state buffers as mapped into this process."""
        n = len(ptrs_A)
        a = (C.c_void_p * n)(*[int(p) for p in ptrs_A])
        b = (C.c_void_p * n)(*[int(p) for p in ptrs_B])
        _check(lib().batl_bind_peers(self._h, a, b))

    def step_part(self, part: int):
        _check(lib().batl_step_part(self._h, int(part)))

    def dt_next_slot(self):
        """int64 view (1 element, on the device) of the running minimum of dt_c: the bit pattern of a positive
        double, whose integer order is the order of the doubles -- what the ranks all-reduce with MIN."""
        import torch
        off = C.c_size_t()
        _check(lib().batl_scalar_offsets(self._h, C.byref(off)))
        return self._bufs[2][off.value:off.value + 8].view(torch.int64)

    def state_pointers(self):
        return self._bufs[0].data_ptr(), self._bufs[1].data_ptr()

    def launch_count(self):
        n = C.c_int64()
        _check(lib().batl_launch_count(self._h, C.byref(n)))
        return n.value


STATIC_MAX_BLOCKS = 4096          # BATL_STATIC_MAX_BLOCKS of include/batl.h


def stable_dt_static(tiles, cell_size, n_blocks, *, gamma, cfl, limiter_beta=2.0, n_order=2, flux_type=0,
                     use_divb_source=1, out_dt, out_warn=None, stream=None):
    """mhd_stable_dt_static of include/batl.h: the CFL time step of a tiled state without a grid object, without a
    scratch buffer and without any allocation (the working data sit in a fixed device array of the library, shared by
    all calls: calls that overlap on the GPU race).  Argument marshalling only.

    tiles: device address (int) or CUDA tensor of [n_blocks][8][12][12][12] doubles with current face ghosts;
    cell_size: CUDA tensor [n_blocks][3]; out_dt: CUDA float64 tensor (1 element); out_warn: CUDA int32 tensor (1
    element) or None; stream: torch stream or None (current stream of the tensors' device).  Enqueues and returns."""
    import torch
    if stream is None:
        stream = torch.cuda.current_stream(out_dt.device)
    ptr = tiles if isinstance(tiles, int) else tiles.data_ptr()
    rc = lib().mhd_stable_dt_static(ptr, cell_size.data_ptr(), int(n_blocks), float(gamma), float(cfl),
                                    float(limiter_beta), int(n_order), int(flux_type), int(use_divb_source),
                                    out_dt.data_ptr(), None if out_warn is None else out_warn.data_ptr(),
                                    stream.cuda_stream)
    if rc < 0:
        raise BatlError(f"batl error {rc}: {lib().batl_static_last_error().decode()}")
