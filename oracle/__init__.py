"""ctypes loader for the CPU oracle (oracle/mhd_oracle.cpp).

TEST INFRASTRUCTURE: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package.  It shares no
code with paper_2501_06717_b200/ and does not import it.

The shared object is compiled on first use with
    g++ -O2 -ffp-contract=off -fopenmp -shared -fPIC
(-ffp-contract=off: no FMA contraction, so the arithmetic is exactly the
expression order written in the source).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "mhd_oracle.cpp")
_LIB = os.path.join(_HERE, "libmhd_oracle.so")
_lib = None

NI, NG, NS, NV = 8, 2, 12, 8


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".{os.getpid()}.tmp"
        cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
               "-o", tmp, _SRC]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        dp, ip = C.POINTER(C.c_double), C.POINTER(C.c_int)
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [ip, dp, dp, ip, dp, C.c_int, ip, dp, C.c_int, C.c_double, C.c_double,
                                 C.c_double, C.c_int, C.c_double, C.c_int, C.c_int, dp, C.c_int,
                                 C.c_double, C.c_double, C.c_double]
        L.orc_set_scheme.argtypes = [C.c_void_p, C.c_int, C.c_int]
        L.orc_set_flux.argtypes = [C.c_void_p, C.c_int]
        L.orc_set_amr.argtypes = [C.c_void_p, C.c_int, C.c_int]
        L.orc_prolong_reads_prolonged.restype = C.c_int64
        L.orc_prolong_reads_prolonged.argtypes = [C.c_void_p]
        L.orc_set_b0_linear.argtypes = [C.c_void_p, dp, dp]
        L.orc_face_flux_type.argtypes = [C.c_int, dp, dp, dp, C.c_double, C.c_int, dp, dp, dp]
        L.orc_free.argtypes = [C.c_void_p]
        L.orc_n_blocks.argtypes = [C.c_void_p]
        L.orc_get_blocks.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_get_neighbors.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_ghost_list.restype = C.c_int64
        L.orc_ghost_list.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_fill_ghosts.argtypes = [C.c_void_p]
        L.orc_set_state.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_set_primitive.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_get_state.argtypes = [C.c_void_p, C.c_void_p, C.c_int]
        L.orc_get_dt_local.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_step.argtypes = [C.c_void_p, C.c_int, dp, dp]
        L.orc_set_threads.argtypes = [C.c_int]
        L.orc_mc_slope.restype = C.c_double
        L.orc_mc_slope.argtypes = [C.c_double, C.c_double, C.c_double]
        L.orc_prim_to_cons.argtypes = [C.c_double, dp, dp]
        L.orc_cons_to_prim.argtypes = [C.c_double, dp, dp]
        L.orc_phys_flux.argtypes = [C.c_int, dp, dp, C.c_double, dp, dp]
        L.orc_face_flux.argtypes = [C.c_int, dp, dp, dp, C.c_double, dp, dp, dp]
        L.orc_dipole_b0.argtypes = [dp, dp, dp]
        L.orc_restrict8.restype = C.c_double
        L.orc_restrict8.argtypes = [dp]
        _lib = L
    return _lib


def _d(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(C.POINTER(C.c_double))


def _i(a):
    a = np.ascontiguousarray(a, dtype=np.int32)
    return a, a.ctypes.data_as(C.POINTER(C.c_int))


class Oracle:
    """One grid + state of the CPU oracle, built from a workloads config dict."""

    def __init__(self, cfg: dict):
        L = lib()
        self.cfg = cfg
        nr, p_nr = _i(cfg["n_root"])
        lo, p_lo = _d(cfg["xyz_min"])
        hi, p_hi = _d(cfg["xyz_max"])
        bc, p_bc = _i(cfg["bc"])
        bp, p_bp = _d(np.asarray(cfg["bc_prim"]).reshape(48))
        regs = cfg["regions"]
        sl, p_sl = _i([[r[0], r[1]] for r in regs] if regs else [[0, 0]])
        rp, p_rp = _d([list(r[2]) for r in regs] if regs else [[0.0] * 6])
        m, p_m = _d(cfg["dipole_m"])
        self._h = L.orc_create(p_nr, p_lo, p_hi, p_bc, p_bp, len(regs), p_sl, p_rp,
                               int(cfg["max_level"]), cfg["gamma"], cfg["cfl"], cfg["limiter_beta"],
                               int(cfg["dt_mode"]), cfg["dt_fixed"], int(cfg["use_divb_source"]),
                               int(cfg["use_b0"]), p_m, int(cfg["use_body"]), cfg["r_body"],
                               cfg["rho_body"], cfg["p_body"])
        L.orc_set_scheme(self._h, int(cfg.get("n_stage", 2)), int(cfg.get("n_order", 2)))
        L.orc_set_flux(self._h, int(cfg.get("flux_type", 0)))
        L.orc_set_amr(self._h, int(cfg.get("prolong_order", 1)), int(cfg.get("flux_correction", 0)))
        self.n_blocks = L.orc_n_blocks(self._h)

    def __del__(self):
        if getattr(self, "_h", None):
            lib().orc_free(self._h)
            self._h = None

    def set_b0_linear(self, c, g):
        """TEST-ONLY background field B0(x) = c + g x (g[a][b] = dB0_a/dx_b); see mhd_oracle.cpp b0_at."""
        c, pc = _d(c)
        g, pg = _d(np.asarray(g, dtype=np.float64).reshape(9))
        lib().orc_set_b0_linear(self._h, pc, pg)

    def prolong_reads_prolonged(self):
        """Number of cells read by the second pass of the second-order prolongation (Q-G4b) that are
        themselves prolonged ghost cells; 0 on a properly nested grid."""
        return int(lib().orc_prolong_reads_prolonged(self._h))

    def blocks(self):
        out = np.zeros((self.n_blocks, 4), dtype=np.int32)
        lib().orc_get_blocks(self._h, out.ctypes.data)
        return out

    def neighbors(self):
        nbr = np.zeros((self.n_blocks, 27, 4), dtype=np.int32)
        dlev = np.zeros((self.n_blocks, 27), dtype=np.int8)
        lib().orc_get_neighbors(self._h, nbr.ctypes.data, dlev.ctypes.data)
        return nbr, dlev

    def ghost_list(self):
        n = lib().orc_ghost_list(self._h, None)
        out = np.zeros((n, 9), dtype=np.int32)
        lib().orc_ghost_list(self._h, out.ctypes.data)
        return out

    def set_state(self, U):
        U = np.ascontiguousarray(U, dtype=np.float64)
        assert U.shape == (self.n_blocks, NV, NI, NI, NI)
        lib().orc_set_state(self._h, U.ctypes.data)

    def set_primitive(self, W):
        W = np.ascontiguousarray(W, dtype=np.float64)
        assert W.shape == (self.n_blocks, NV, NI, NI, NI)
        lib().orc_set_primitive(self._h, W.ctypes.data)

    def get_state(self, with_ghost=False):
        n = NS if with_ghost else NI
        out = np.zeros((self.n_blocks, NV, n, n, n))
        lib().orc_get_state(self._h, out.ctypes.data, int(with_ghost))
        return out

    def get_dt_local(self):
        out = np.zeros((self.n_blocks, NI, NI, NI))
        lib().orc_get_dt_local(self._h, out.ctypes.data)
        return out

    def fill_ghosts(self):
        lib().orc_fill_ghosts(self._h)

    def step(self, n_steps=1):
        """Returns (warning bitmask, t, dt_last)."""
        t, dt = C.c_double(0.0), C.c_double(0.0)
        w = lib().orc_step(self._h, int(n_steps), C.byref(t), C.byref(dt))
        return w, t.value, dt.value


# ---- unit-level wrappers used by the pins --------------------------------------
def mc_slope(dm, dp, beta=2.0):
    return lib().orc_mc_slope(float(dm), float(dp), float(beta))


def prim_to_cons(W, gamma=5.0 / 3.0):
    W, pw = _d(W)
    U = np.zeros(8)
    lib().orc_prim_to_cons(gamma, pw, U.ctypes.data_as(C.POINTER(C.c_double)))
    return U


def cons_to_prim(U, gamma=5.0 / 3.0):
    U, pu = _d(U)
    W = np.zeros(8)
    lib().orc_cons_to_prim(gamma, pu, W.ctypes.data_as(C.POINTER(C.c_double)))
    return W


def phys_flux(d, W, B0f=(0, 0, 0), gamma=5.0 / 3.0):
    W, pw = _d(W)
    B0, pb = _d(B0f)
    F, U = np.zeros(8), np.zeros(8)
    dp = C.POINTER(C.c_double)
    lib().orc_phys_flux(int(d), pw, pb, gamma, F.ctypes.data_as(dp), U.ctypes.data_as(dp))
    return F, U


def face_flux(d, WL, WR, B0f=(0, 0, 0), gamma=5.0 / 3.0, flux_type=0):
    WL, pl = _d(WL)
    WR, pr = _d(WR)
    B0, pb = _d(B0f)
    F = np.zeros(8)
    bn, c = C.c_double(0), C.c_double(0)
    lib().orc_face_flux_type(int(d), pl, pr, pb, gamma, int(flux_type), F.ctypes.data_as(C.POINTER(C.c_double)),
                             C.byref(bn), C.byref(c))
    return F, bn.value, c.value


def dipole_b0(m, x):
    m, pm = _d(m)
    x, px = _d(x)
    B = np.zeros(3)
    lib().orc_dipole_b0(pm, px, B.ctypes.data_as(C.POINTER(C.c_double)))
    return B


def restrict8(a):
    a, pa = _d(a)
    return lib().orc_restrict8(pa)


def set_threads(n):
    lib().orc_set_threads(int(n))


def max_threads():
    return lib().orc_max_threads()
