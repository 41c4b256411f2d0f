"""Pins for the oracle's grid builder, neighbour table and ghost fill (CPU only).

Every expected value here comes from the paper (cited), from a closed form, or
from a hand / coordinate-based enumeration that does not call the oracle.
"""
import itertools

import numpy as np
import pytest

import workloads as wl


def _dir(d):
    return (d[0] + 1) + 3 * (d[1] + 1) + 9 * (d[2] + 1)


# ------------------------------------------------------------------ leaf counts
def test_leaf_counts_table2(orc):
    # PAPER.md Table 2 (L257-337) / L185: 2x2x2 roots with one octant refined gives
    # 15 blocks, 4x4x4 roots with [-32,0]^3 refined gives 15*2^3 = 120.
    assert orc.Oracle(wl.fast_wave((2, 2, 2))).n_blocks == 15
    assert orc.Oracle(wl.fast_wave((4, 4, 4))).n_blocks == 120
    from util import golden
    gv = golden()                                        # the same counts as printed in the paper
    for n in (2, 4, 8):
        assert orc.Oracle(wl.fast_wave((n, n, n))).n_blocks == gv[f"blocks.roots_{n}"] == 15 * n ** 3 // 8
    assert 1920 * 2 ** 9 * 1000 // 10 ** 6 == gv["cells.largest_run_millions"]


def test_leaf_count_config3(orc):
    # BASELINE.json configs[2]: 8x4x4 roots, blocks intersecting |x|<0.25 refined:
    # root columns ix in {3,4} -> 32 roots -> 96 coarse + 256 fine (SURVEY Q-O3)
    o = orc.Oracle(wl.brio_wu_amr())
    blk = o.blocks()
    assert o.n_blocks == 352
    assert (blk[:, 0] == 0).sum() == 96 and (blk[:, 0] == 1).sum() == 256
    fine_roots = set((b[1] >> 1, b[2] >> 1, b[3] >> 1) for b in blk if b[0] == 1)
    assert fine_roots == set((ix, iy, iz) for ix in (3, 4) for iy in range(4) for iz in range(4))


def test_magnetosphere_grid(orc):
    # 3,788 blocks of 8^3, ~2 M cells; our synthetic stand-in with
    # radii (96,48,24) must be within 1% of that and the body must sit in finest blocks
    cfg = wl.magnetosphere()
    o = orc.Oracle(cfg)
    assert abs(o.n_blocks - 3788) / 3788 < 0.01
    blk = o.blocks()
    assert blk[:, 0].max() == 4 and blk[:, 0].min() == 1
    for b in blk:
        x, y, z = wl.cell_centres(cfg, b)
        d = wl.cell_size(cfg, b[0])
        lo = np.array([x[0], y[0], z[0]]) - d / 2
        hi = np.array([x[-1], y[-1], z[-1]]) + d / 2
        dist = np.sqrt((np.maximum(0, np.maximum(lo, -hi)) ** 2).sum())
        if dist < cfg["r_body"] + 2 * d.max():
            assert b[0] == 4


# --------------------------------------------------------------- ordering (Q-O1)
def test_morton_order_15_leaf(orc):
    blk = orc.Oracle(wl.fast_wave((2, 2, 2))).blocks()
    expect = []
    for root in range(8):
        rx, ry, rz = root & 1, (root >> 1) & 1, root >> 2
        if (rx, ry, rz) == (0, 0, 0):           # [-32,0]^3 is root (0,0,0)
            for c in range(8):
                expect.append((1, c & 1, (c >> 1) & 1, c >> 2))
        else:
            expect.append((0, rx, ry, rz))
    assert [tuple(b) for b in blk] == expect


def test_uniform_periodic_neighbours_closed_form(orc):
    n = (4, 3, 2)
    cfg = wl.random_uniform(n)
    o = orc.Oracle(cfg)
    blk = o.blocks()
    ids = {tuple(b[1:]): i for i, b in enumerate(blk)}
    # natural root order
    assert [tuple(b) for b in blk] == [(0, i, j, k) for k in range(n[2]) for j in range(n[1]) for i in range(n[0])]
    nbr, dlev = o.neighbors()
    assert (dlev == 0).all()
    for b, (_, I, J, K) in enumerate(blk):
        for d in itertools.product((-1, 0, 1), repeat=3):
            e = ids[((I + d[0]) % n[0], (J + d[1]) % n[1], (K + d[2]) % n[2])]
            assert nbr[b, _dir(d), 0] == e and (nbr[b, _dir(d), 1:] == -1).all()


def test_two_root_hand_enumeration(orc):
    # domain [0,2]x[0,1]x[0,1], roots (0,0,0) and (1,0,0); root 0 refined; all faces float.
    cfg = wl._base("two", (2, 1, 1), (0, 0, 0), (2, 1, 1), bc=(1,) * 6,
                   regions=[(wl.SHAPE_BOX, 1, (0, 0, 0, 1, 1, 1))], max_level=1)
    o = orc.Oracle(cfg)
    blk = [tuple(b) for b in o.blocks()]
    # 8 children of root 0 in child-digit order, then root 1
    assert blk == [(1, c & 1, (c >> 1) & 1, c >> 2) for c in range(8)] + [(0, 1, 0, 0)]
    nbr, dlev = o.neighbors()
    coarse = 8
    # coarse block: -x face neighbour is finer: the 4 children with ox=1, y fastest then z
    assert dlev[coarse, _dir((-1, 0, 0))] == -1
    assert list(nbr[coarse, _dir((-1, 0, 0))]) == [1, 3, 5, 7]
    # everything else of the coarse block is outside the (non-periodic) domain
    for d in itertools.product((-1, 0, 1), repeat=3):
        if d not in ((0, 0, 0), (-1, 0, 0)):
            assert dlev[coarse, _dir(d)] == -100 and (nbr[coarse, _dir(d)] == -1).all()
    assert dlev[coarse, 13] == 0 and nbr[coarse, 13, 0] == coarse
    # fine child 1 = (1,0,0) [ox=1,oy=0,oz=0]: +x is the coarse root; +y is child 3; -x child 0
    assert dlev[1, _dir((1, 0, 0))] == 1 and nbr[1, _dir((1, 0, 0)), 0] == coarse
    assert dlev[1, _dir((0, 1, 0))] == 0 and nbr[1, _dir((0, 1, 0)), 0] == 3
    assert dlev[1, _dir((-1, 0, 0))] == 0 and nbr[1, _dir((-1, 0, 0)), 0] == 0
    assert dlev[1, _dir((1, 1, 0))] == 1 and nbr[1, _dir((1, 1, 0)), 0] == coarse  # edge lies in coarse face
    assert dlev[1, _dir((1, 1, 1))] == 1 and nbr[1, _dir((1, 1, 1)), 0] == coarse
    assert dlev[1, _dir((0, -1, 0))] == -100
    assert dlev[1, _dir((0, 1, 1))] == 0 and nbr[1, _dir((0, 1, 1)), 0] == 7


def test_nesting_is_enforced(orc):
    # 4x1x1 roots; only root 0 asked to level 2.  Q-O2: root 1 must go to level 1.
    reg = [(wl.SHAPE_BOX, 2, (0, 0, 0, 1, 1, 1))]
    flo = wl._base("n", (4, 1, 1), (0, 0, 0), (4, 1, 1), bc=(1,) * 6, regions=reg, max_level=2)
    assert orc.Oracle(flo).n_blocks == 64 + 8 + 1 + 1
    per = wl._base("n", (4, 1, 1), (0, 0, 0), (4, 1, 1), regions=reg, max_level=2)
    assert orc.Oracle(per).n_blocks == 64 + 8 + 1 + 8     # root 3 touches root 0 through the wrap


def test_edge_dlev_consistency(orc):
    # every listed neighbour really is at the stated level, and relations are mutual for faces
    o = orc.Oracle(wl.fast_wave((2, 2, 2)))
    blk = o.blocks()
    nbr, dlev = o.neighbors()
    for b in range(o.n_blocks):
        for dr in range(27):
            for q in range(4):
                n = nbr[b, dr, q]
                if n >= 0:
                    assert blk[b, 0] - blk[n, 0] == dlev[b, dr]


# ------------------------------------------------------------------- ghost fill
def _linear(x, y, z):
    return 1.0 + 2.0 * x - 3.0 * y + 5.0 * z        # exact in fp64 for our dyadic coordinates


def _expected_ghost_value(cfg, blocks, b, i, j, k):
    """Coordinate-based re-derivation (no index arithmetic shared with the oracle):
    centre of the ghost cell -> wrap / clamp into the domain -> block containing
    the point -> value by level relation."""
    lev = blocks[b][0]
    d = wl.cell_size(cfg, lev)
    lo, hi = np.array(cfg["xyz_min"]), np.array(cfg["xyz_max"])
    c = lo + (8 * np.array(blocks[b][1:]) + np.array([i, j, k]) + 0.5) * d
    for a in range(3):
        if c[a] < lo[a] or c[a] > hi[a]:
            face = 2 * a + (1 if c[a] > hi[a] else 0)
            if cfg["bc"][face] == wl.BC_PERIODIC:
                c[a] = lo[a] + (c[a] - lo[a]) % (hi[a] - lo[a])
            elif cfg["bc"][face] == wl.BC_FLOAT:
                c[a] = min(max(c[a], lo[a] + d[a] / 2), hi[a] - d[a] / 2)
            else:
                return None
    for blk in blocks:                    # which leaf contains the point?
        size = 8 * wl.cell_size(cfg, blk[0])
        blo = lo + np.array(blk[1:]) * size
        if np.all(c > blo) and np.all(c < blo + size):
            if blk[0] <= lev - 1:         # coarser: value of the coarse cell containing the point
                dc = wl.cell_size(cfg, blk[0])
                cc = lo + (np.floor((c - lo) / dc) + 0.5) * dc
                return _linear(*cc)
            return _linear(*c)            # same level: copy; finer: mean of a linear field
    raise AssertionError("point not covered")


@pytest.mark.parametrize("cfgname", ["fast15", "two_float"])
def test_ghost_values_restriction_prolongation_copy(orc, cfgname):
    if cfgname == "fast15":
        cfg = wl.fast_wave((2, 2, 2))     # periodic, 15 leaves, two levels
    else:
        cfg = wl._base("two", (2, 1, 1), (0, 0, 0), (2, 1, 1), bc=(1,) * 6,
                       regions=[(wl.SHAPE_BOX, 1, (0, 0, 0, 1, 1, 1))], max_level=1)
    o = orc.Oracle(cfg)
    blocks = [tuple(int(v) for v in b) for b in o.blocks()]
    U = np.zeros((o.n_blocks, 8, 8, 8, 8))
    for b, blk in enumerate(blocks):
        x, y, z = wl.cell_centres(cfg, blk)
        f = _linear(x[None, None, :], y[None, :, None], z[:, None, None])
        for v in range(8):
            U[b, v] = f + 1000.0 * v
    o.set_state(U)
    G = o.get_state(with_ghost=True)
    rng = np.random.default_rng(7)
    cells = [(i, j, k) for k in range(-2, 10) for j in range(-2, 10) for i in range(-2, 10)
             if not (0 <= i < 8 and 0 <= j < 8 and 0 <= k < 8)]
    for b in range(o.n_blocks):
        sel = cells if b in (0, 7, o.n_blocks - 1) else [cells[q] for q in rng.choice(len(cells), 150, replace=False)]
        for (i, j, k) in sel:
            e = _expected_ghost_value(cfg, blocks, b, i, j, k)
            for v in (0, 5):
                assert G[b, v, k + 2, j + 2, i + 2] == e + 1000.0 * v, (b, i, j, k)


def test_L115_worked_example_and_L146_sizes(orc):
    # block B is the +x neighbour of A: A's cells nI+1, nI+2 (0-based 8, 9)
    # take B's cells 1, 2 (0-based 0, 1), same j, k.
    cfg = wl.random_uniform((3, 3, 3))
    o = orc.Oracle(cfg)
    gl = o.ghost_list()
    nbr, _ = o.neighbors()
    A = 13
    Bx = nbr[A, _dir((1, 0, 0)), 0]
    rows = gl[(gl[:, 0] == A) & (gl[:, 3] >= 8) & (gl[:, 1] >= 0) & (gl[:, 1] < 8) & (gl[:, 2] >= 0) & (gl[:, 2] < 8)]
    assert len(rows) == 8 * 8 * 2                                   # L146: face = nJ nK nG cells
    assert (rows[:, 4] == 0).all() and (rows[:, 5] == Bx).all()
    assert (rows[:, 8] == rows[:, 3] - 8).all() and (rows[:, 6] == rows[:, 1]).all() and (rows[:, 7] == rows[:, 2]).all()
    # L146 sizes with nI=8, nG=2, nV=8: face 1024, edge 256, corner 64 reals = 128 / 32 / 8 cells
    a = gl[gl[:, 0] == A]
    nout = ((a[:, 1:4] < 0) | (a[:, 1:4] > 7)).sum(axis=1)
    assert (nout == 1).sum() == 6 * 128 and (nout == 2).sum() == 12 * 32 and (nout == 3).sum() == 8 * 8
    assert len(a) == 1216
    # the paper's own figures (tests/golden): corner nG^3 nV = 64 reals, face nI nJ nG nV = 1,600 reals at nI = 10
    from util import golden
    gv = golden()
    nG, nV = 2, 8
    assert nG ** 3 * nV == gv["message.corner_reals"] == 8 * nV          # 8 cells per corner here too
    assert 10 * 10 * nG * nV == gv["message.face_reals"]
    assert 128 * nV == gv["message.face_reals"] * 8 * 8 // (10 * 10)     # scaled to 8^3 blocks: 1,024 reals


def test_L146_coarser_neighbour_sizes(orc):
    # L146: towards a coarser neighbour the message is divided by 4 (face) or 2 (edge).
    o = orc.Oracle(wl._base("two", (2, 1, 1), (0, 0, 0), (2, 1, 1), bc=(1,) * 6,
                            regions=[(wl.SHAPE_BOX, 1, (0, 0, 0, 1, 1, 1))], max_level=1))
    gl = o.ghost_list()
    coarse = 8
    # restricted cells of the coarse block's -x FACE region (edge/corner regions clamp into it too)
    r = gl[(gl[:, 0] == coarse) & (gl[:, 4] == 1) & (gl[:, 1] >= 0) & (gl[:, 1] < 8) & (gl[:, 2] >= 0) & (gl[:, 2] < 8)]
    per_src = {s: (r[:, 5] == s).sum() for s in (1, 3, 5, 7)}
    # the coarse -x face ghost (8x8x2 = 128 cells) is shared by 4 fine blocks: 128/4 each
    assert all(n == 32 for n in per_src.values())
    from util import golden
    assert 128 // 32 == golden()["message.coarser_face_divisor"]
    # and each restricted cell points at the lowest-index fine cell of its 2x2x2 group
    assert (r[:, 6:9] % 2 == 0).all()
    # fine block 1: +x face ghosts (128 fine cells) are prolonged from 4x4x1 coarse cells
    p = gl[(gl[:, 0] == 1) & (gl[:, 4] == 2) & (gl[:, 3] >= 8) & (gl[:, 1] >= 0) & (gl[:, 1] < 8) & (gl[:, 2] >= 0) & (gl[:, 2] < 8)]
    assert len(p) == 128 and len(set(map(tuple, p[:, 5:9]))) == 16
    assert (p[:, 8] == 0).all()


def test_fixed_boundary_and_float(orc):
    cfg = wl.magnetosphere()
    o = orc.Oracle(cfg)
    blk = o.blocks()
    W = wl.initial_primitive(cfg, blk)
    W[:, 0] += 0.25 * np.arange(o.n_blocks)[:, None, None, None]     # make blocks distinguishable
    o.set_primitive(W)
    G = o.get_state(with_ghost=True)
    P = o.get_state()
    nx = cfg["n_root"][0] << 1
    b = next(i for i, q in enumerate(blk) if q[0] == 1 and q[1] == nx - 1)     # touches +x (fixed)
    sw = wl.SW_RHO, wl.SW_UX, wl.SW_BZ, wl.SW_P
    # closed form of eq. (5), for the solar-wind state
    e = sw[3] / (cfg["gamma"] - 1) + 0.5 * sw[0] * sw[1] ** 2 + 0.5 * sw[2] ** 2
    assert np.all(G[b, 0, 2:10, 2:10, 10:] == sw[0])
    assert np.all(G[b, 1, 2:10, 2:10, 10:] == sw[0] * sw[1])
    assert np.all(G[b, 6, 2:10, 2:10, 10:] == sw[2])
    assert np.allclose(G[b, 7, 2:10, 2:10, 10:], e, rtol=1e-15)
    b = next(i for i, q in enumerate(blk) if q[0] == 1 and q[1] == 0)          # touches -x (float)
    for v in range(8):
        assert np.all(G[b, v, 2:10, 2:10, 0] == P[b, v, :, :, 0])
        assert np.all(G[b, v, 2:10, 2:10, 1] == P[b, v, :, :, 0])


def test_restriction_order_and_uniform_exactness(orc):
    # Q-G3 pairwise order reproduces a constant exactly and equals the exact mean for dyadic data
    a = np.array([1.0, 3.0, 5.0, 7.0, 9.0, 11.0, 13.0, 15.0])
    assert orc.restrict8(a) == 8.0
    c = 0.1 + 0.2          # not exactly representable
    assert orc.restrict8(np.full(8, c)) == c
    # order sensitivity: (((a0+a1)+(a2+a3))+((a4+a5)+(a6+a7)))/8 with a cancellation pattern
    a = np.array([1e16, 1.0, -1e16, 1.0, 0, 0, 0, 0])
    assert orc.restrict8(a) == ((1e16 + 1.0) + (-1e16 + 1.0)) * 0.125


def test_uniform_state_ghosts_bit_identical(orc):
    for cfg in (wl.fast_wave((2, 2, 2)), wl.brio_wu_amr()):
        cfg = wl.uniform_state(cfg)
        o = orc.Oracle(cfg)
        o.set_primitive(wl.initial_primitive(cfg, o.blocks()))
        G = o.get_state(with_ghost=True)
        for v in range(8):
            assert np.all(G[:, v] == G[0, v, 5, 5, 5])
