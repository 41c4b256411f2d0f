"""Seeded synthetic workloads shared by the oracle tests and the CUDA path.

This module holds NONE of the method's arithmetic: it only describes grids
(plain dictionaries) and produces initial fields on cell centres, as PRIMITIVE
variables (rho, u, B1, p) and -- for callers of the C ABI, whose input is the
conserved state -- in the conserved form that PAPER.md eq. (5), defines
(``prim_to_cons``: input formatting, not a step of the time integration).  The
block tree, the ghost fill, the primitive recovery and the solver are implemented
separately by ``oracle/`` and by ``paper_2501_06717_b200/``; neither imports the
other.

The five configurations are the ones BASELINE.json lists (SURVEY.md §8(d)
"Synthetic inputs").  They stand in for the paper's workloads (fast wave,
PAPER.md L185/L339-343, and the magnetosphere run, L389-391), whose input
files are not available; all fields are generated from closed forms plus
``numpy.random.default_rng`` streams keyed by (seed, level, I, J, K) of each
block, so the values do not depend on the block order.

Geometry contract (include/batl.h): a block is (level, I, J, K); its cell size
is D_a = (max_a - min_a) / (8 n_root_a) * 2**-level and cell centres are at
x_a = min_a + (8 I_a + i + 1/2) D_a, i = 0..7.
"""
from __future__ import annotations

import math

import numpy as np

NI = 8          # cells per block and axis (n_I = n_J = n_K = 8)
NV = 8          # rho, ux, uy, uz, Bx, By, Bz, p (primitive order)
BASE_SEED = 20250106

BC_PERIODIC, BC_FLOAT, BC_FIXED = 0, 1, 2
SHAPE_ALL, SHAPE_BOX, SHAPE_SPHERE = 0, 1, 2
DT_GLOBAL, DT_LOCAL, DT_FIXED = 0, 1, 2


def _base(name, n_root, lo, hi, **kw):
    cfg = dict(
        name=name,
        n_root=tuple(int(n) for n in n_root),
        xyz_min=tuple(float(x) for x in lo),
        xyz_max=tuple(float(x) for x in hi),
        bc=(BC_PERIODIC,) * 6,
        bc_prim=np.zeros((6, NV)),
        regions=[],               # list of (shape, level, (p0..p5))
        max_level=0,
        gamma=5.0 / 3.0,
        cfl=0.8,
        limiter_beta=2.0,
        n_stage=2,                # 1: one-stage scheme
        n_order=2,                # 1: piecewise-constant face states (L86 nOrder)
        flux_type=0,              # 1: HLL-type "Linde" flux (L343, Q-F4)
        prolong_order=1,          # 2: second-order limited prolongation (Q-G4b)
        flux_correction=0,        # 1: conservative flux correction at resolution changes (Q-G6b)
        dt_mode=DT_GLOBAL,
        dt_fixed=0.0,
        use_divb_source=1,
        use_b0=0,
        dipole_m=(0.0, 0.0, 0.0),
        use_body=0,
        r_body=0.0,
        rho_body=1.0,
        p_body=-1.0,              # <= 0: pressure floats at the body
        n_steps=10,
        seed=BASE_SEED,
        field="uniform",
        field_params={},
    )
    cfg.update(kw)
    return cfg


# ----------------------------------------------------------------------------
# the five BASELINE.json configurations
# ----------------------------------------------------------------------------
def alfven(n_root=(2, 2, 2), amplitude=0.1, n_steps=10, **kw):
    """configs[0]: circularly polarised Alfven wave along x on [0,1]^3."""
    hi = tuple(n / n_root[0] for n in n_root)      # cubic cells, x length 1
    return _base("alfven", n_root, (0, 0, 0), hi, n_steps=n_steps,
                 seed=BASE_SEED + 1, field="alfven",
                 field_params=dict(amplitude=amplitude, rho=1.0, p=0.1, bx=1.0), **kw)


def orszag_tang(n_root=(8, 8, 8), n_steps=100, **kw):
    """configs[1]: Orszag-Tang-type vortex extended along z on [0,2pi]^3."""
    two_pi = 2.0 * math.pi
    return _base("orszag_tang_z", n_root, (0, 0, 0), (two_pi,) * 3, n_steps=n_steps,
                 seed=BASE_SEED + 2, field="orszag_tang",
                 field_params=dict(perturb=1e-3), **kw)


def brio_wu_amr(n_steps=200, **kw):
    """configs[2]: Brio-Wu shock tube on a two-level grid; |x|<0.25 refined."""
    bc = (BC_FLOAT, BC_FLOAT, BC_PERIODIC, BC_PERIODIC, BC_PERIODIC, BC_PERIODIC)
    regions = [(SHAPE_BOX, 1, (-0.25, -1e30, -1e30, 0.25, 1e30, 1e30))]
    return _base("brio_wu_amr", (8, 4, 4), (-1, -0.5, -0.5), (1, 0.5, 0.5), bc=bc,
                 regions=regions, max_level=1, n_steps=n_steps,
                 seed=BASE_SEED + 3, field="brio_wu", **kw)


def random_uniform(n_root=(16, 16, 16), n_steps=50, **kw):
    """configs[3]: seeded Gaussian perturbations on a uniform periodic grid.

    The throughput sweep uses n_root = 8^3, 16*8*8, 16*16*8, 16^3, 32*16*16,
    32*32*16, 32^3 (512 ... 32768 blocks); 16^3 = 4096 blocks is the bench case.
    """
    return _base("random_uniform", n_root, (0, 0, 0), tuple(float(n) for n in n_root),
                 n_steps=n_steps, seed=BASE_SEED + 4, field="random", **kw)


# code units of configs[4]: length R_E, rho in m_p/cm^3, u in km/s
#   => B unit 0.0458463 nT, p unit 1.67262e-6 nPa
SW_RHO, SW_UX, SW_BZ, SW_P = 5.0, -400.0, -109.060, 4127.20
DIPOLE_MZ = -678354.0     # 31,100 nT R_E^3 in code units, moment along -z


def magnetosphere(radii=(96.0, 48.0, 24.0), n_steps=100, **kw):
    """configs[4]: magnetosphere-like run, 4 levels, B0 dipole, body, local dt."""
    bc = (BC_FLOAT, BC_FIXED, BC_FLOAT, BC_FLOAT, BC_FLOAT, BC_FLOAT)
    bc_prim = np.zeros((6, NV))
    bc_prim[1] = (SW_RHO, SW_UX, 0, 0, 0, 0, SW_BZ, SW_P)       # +x face: solar wind
    regions = [(SHAPE_ALL, 1, (0,) * 6)]
    for lev, r in enumerate(radii, start=2):
        regions.append((SHAPE_SPHERE, lev, (0.0, 0.0, 0.0, float(r), 0.0, 0.0)))
    return _base("magnetosphere", (4, 4, 4), (-224, -128, -128), (32, 128, 128), bc=bc,
                 bc_prim=bc_prim, regions=regions, max_level=4, cfl=0.6,
                 dt_mode=DT_LOCAL, use_b0=1, dipole_m=(0.0, 0.0, DIPOLE_MZ),
                 use_body=1, r_body=2.5, rho_body=28.0, n_steps=n_steps,
                 seed=BASE_SEED + 5, field="magnetosphere",
                 field_params=dict(r_taper=8.0), **kw)


CONFIGS = {0: alfven, 1: orszag_tang, 2: brio_wu_amr, 3: random_uniform, 4: magnetosphere}


# ----------------------------------------------------------------------------
# extra small grids used by the pins and parity tests
# ----------------------------------------------------------------------------
def fast_wave(n_root=(2, 2, 2), refine_octant=True, amplitude_scale=1.0, **kw):
    """The paper's fast-wave set-up (eq. 6 as decoded in
    SURVEY.md Appendix A): domain [-32,32]^3, octant [-32,0]^3 refined 2:1."""
    regions = [(SHAPE_BOX, 1, (-32.0, -32.0, -32.0, 0.0, 0.0, 0.0))] if refine_octant else []
    return _base("fast_wave", n_root, (-32,) * 3, (32,) * 3, regions=regions,
                 max_level=1 if refine_octant else 0, seed=BASE_SEED + 6, field="fast_wave",
                 field_params=dict(scale=amplitude_scale), **kw)


def uniform_state(cfg, prim=(1.3, 0.2, -0.1, 0.05, 0.7, -0.4, 0.3, 0.9)):
    """Same grid as cfg, but a constant primitive state."""
    out = dict(cfg)
    out["field"] = "uniform"
    out["field_params"] = dict(prim=tuple(prim))
    return out


# ----------------------------------------------------------------------------
# geometry helpers (no physics)
# ----------------------------------------------------------------------------
def cell_size(cfg, level):
    return np.array([(cfg["xyz_max"][a] - cfg["xyz_min"][a]) / (NI * cfg["n_root"][a])
                     for a in range(3)]) * 2.0 ** (-int(level))


def cell_centres(cfg, blk):
    """x[i], y[j], z[k] cell-centre coordinates of block (level, I, J, K)."""
    level = int(blk[0])
    d = cell_size(cfg, level)
    idx = np.arange(NI) + 0.5
    return [cfg["xyz_min"][a] + (NI * int(blk[1 + a]) + idx) * d[a] for a in range(3)]


def _block_rng(cfg, blk):
    return np.random.default_rng([int(cfg["seed"])] + [int(v) for v in blk])


def initial_primitive(cfg, blocks):
    """Primitive initial state W[nB][8 vars][k][j][i] for the given block list.

    blocks: int array [nB][4] = (level, I, J, K) in the caller's block order.
    """
    blocks = np.asarray(blocks, dtype=np.int64).reshape(-1, 4)
    nb = blocks.shape[0]
    w = np.zeros((nb, NV, NI, NI, NI))
    kind = cfg["field"]
    fp = cfg["field_params"]
    for b in range(nb):
        blk = blocks[b]
        x, y, z = cell_centres(cfg, blk)
        X = x[None, None, :] + 0 * y[None, :, None] + 0 * z[:, None, None]
        Y = 0 * X + y[None, :, None]
        Z = 0 * X + z[:, None, None]
        wb = w[b]
        if kind == "uniform":
            prim = fp.get("prim", (1.0, 0, 0, 0, 0, 0, 0, 1.0))
            for v in range(NV):
                wb[v] = prim[v]
        elif kind == "alfven":
            a, rho, p, bx = fp["amplitude"], fp["rho"], fp["p"], fp["bx"]
            ph = 2.0 * math.pi * X
            by, bz = a * np.cos(ph), a * np.sin(ph)
            wb[0], wb[7], wb[4] = rho, p, bx
            wb[5], wb[6] = by, bz
            wb[2], wb[3] = -by / math.sqrt(rho), -bz / math.sqrt(rho)
        elif kind == "orszag_tang":
            rng = _block_rng(cfg, blk)
            wb[0] = 25.0 / (36.0 * math.pi)
            wb[7] = 5.0 / (12.0 * math.pi)
            wb[1], wb[2], wb[3] = -np.sin(Y), np.sin(X), 0.0
            wb[4] = -np.sin(Y) / math.sqrt(4.0 * math.pi)
            wb[5] = np.sin(2.0 * X) / math.sqrt(4.0 * math.pi)
            wb[1:4] += rng.uniform(-fp["perturb"], fp["perturb"], size=(3, NI, NI, NI))
        elif kind == "brio_wu":
            left = X < 0.0
            wb[0] = np.where(left, 1.0, 0.125)
            wb[7] = np.where(left, 1.0, 0.1)
            wb[4] = 0.75
            wb[5] = np.where(left, 1.0, -1.0)
        elif kind == "random":
            rng = _block_rng(cfg, blk)
            n = np.clip(rng.standard_normal(size=(NV, NI, NI, NI)), -4.0, 4.0)
            s = 1.0 / math.sqrt(2.0)
            wb[0] = 1.0 + 0.05 * n[0]
            wb[7] = 1.0 + 0.05 * n[7]
            wb[1:4] = 0.1 * n[1:4]
            wb[4] = s + 0.1 * n[4]
            wb[5] = s + 0.1 * n[5]
            wb[6] = 0.1 * n[6]
        elif kind == "fast_wave":
            # V0 + V1 cos(k x), k = pi/16
            sc = fp["scale"]
            c = sc * np.cos(math.pi / 16.0 * X)
            wb[0] = 1.0 + 0.1 * c
            wb[1] = 0.005 * c
            wb[5] = 0.04 + 0.004 * c
            wb[7] = 0.00054 + 0.00009 * c
        elif kind == "magnetosphere":
            r = np.sqrt(X * X + Y * Y + Z * Z)
            rb, rt = cfg["r_body"], fp["r_taper"]
            taper = np.clip((r - rb) / (rt - rb), 0.0, 1.0)
            wb[0] = np.where(r < rb, cfg["rho_body"], SW_RHO)
            wb[1] = SW_UX * taper
            wb[6] = SW_BZ
            wb[7] = SW_P
        else:
            raise ValueError(f"unknown field {kind!r}")
    return w


def prim_to_cons(W, gamma):
    """Input formatting for the C ABI (batl_set_state takes conserved variables): the conserved
    form (rho, rho u, B1, e) of primitive fields W[nB][8][...] by the definition of the energy
    density, eq. (5), L179-181.  Host numpy; not part of the time step."""
    W = np.asarray(W, dtype=np.float64)
    U = np.empty_like(W)
    U[:, 0] = W[:, 0]
    U[:, 1:4] = W[:, 0:1] * W[:, 1:4]
    U[:, 4:7] = W[:, 4:7]
    U[:, 7] = W[:, 7] / (gamma - 1.0) + 0.5 * W[:, 0] * (W[:, 1:4] ** 2).sum(axis=1) + 0.5 * (W[:, 4:7] ** 2).sum(axis=1)
    return U


def initial_conserved(cfg, blocks):
    """Conserved initial state U[nB][8][k][j][i] of the configuration (see prim_to_cons)."""
    return prim_to_cons(initial_primitive(cfg, blocks), cfg["gamma"])
