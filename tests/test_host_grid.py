"""Host logic of the library vs the oracle (CPU only): block order, neighbour table
and expanded ghost lists must be BIT-EXACT (BASELINE.json north_star), and the C-ABI
library must load and export every symbol include/batl.h declares."""
import ctypes
import os
import re

import numpy as np
import pytest

import workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _mixed_bc_amr():
    # refined corner region that touches float, fixed and periodic faces at once
    cfg = wl.fast_wave((2, 2, 2))
    cfg = dict(cfg)
    cfg["bc"] = (wl.BC_FLOAT, wl.BC_FIXED, wl.BC_FLOAT, wl.BC_FLOAT, wl.BC_PERIODIC, wl.BC_PERIODIC)
    bp = np.zeros((6, 8))
    bp[1] = (2.0, 0.1, 0.2, 0.3, 0.4, 0.5, 0.6, 0.7)
    cfg["bc_prim"] = bp
    return cfg


def _three_level():
    cfg = dict(wl.fast_wave((2, 2, 2)))
    cfg["regions"] = [(wl.SHAPE_BOX, 1, (-32.0, -32.0, -32.0, 0.0, 0.0, 0.0)),
                      (wl.SHAPE_SPHERE, 3, (-30.0, -30.0, -30.0, 3.0, 0.0, 0.0))]
    cfg["max_level"] = 3
    cfg["bc"] = (wl.BC_FLOAT, wl.BC_FLOAT, wl.BC_PERIODIC, wl.BC_PERIODIC, wl.BC_FIXED, wl.BC_FIXED)
    return cfg


CASES = {
    "alfven_2x2x2": lambda: wl.alfven(),
    "uniform_1x1x1": lambda: wl.random_uniform((1, 1, 1)),
    "uniform_2x1x3": lambda: wl.random_uniform((2, 1, 3)),
    "uniform_4x3x2": lambda: wl.random_uniform((4, 3, 2)),
    "fast_wave_15": lambda: wl.fast_wave((2, 2, 2)),
    "fast_wave_120": lambda: wl.fast_wave((4, 4, 4)),
    "brio_wu_amr": lambda: wl.brio_wu_amr(),
    "mixed_bc_amr": _mixed_bc_amr,
    "three_level": _three_level,
    "magnetosphere": lambda: wl.magnetosphere(),
}


def test_library_exports_every_declared_symbol():
    import paper_2501_06717_b200 as batl
    L = batl.lib()
    header = open(os.path.join(ROOT, "include", "batl.h")).read()
    declared = set(re.findall(r"^\s*(?:int|void|const char\*)\s+(\w+)\s*\(", header, flags=re.M))
    assert declared, "no prototypes found in include/batl.h"
    assert declared == set(batl.EXPORTS)
    for name in declared:
        assert getattr(L, name) is not None
    # plain C symbols, no C++ mangling
    raw = ctypes.CDLL(batl._build.LIB)
    for name in declared:
        getattr(raw, name)


@pytest.mark.parametrize("name", sorted(CASES))
def test_tables_bit_exact_vs_oracle(orc, name):
    import paper_2501_06717_b200 as batl
    cfg = CASES[name]()
    o = orc.Oracle(cfg)
    g = batl.Grid(cfg)
    assert g.n_blocks == o.n_blocks
    assert np.array_equal(g.blocks(), o.blocks())
    nbr_o, dlev_o = o.neighbors()
    nbr_g, dlev_g = g.neighbors()
    assert np.array_equal(dlev_g, dlev_o)
    assert np.array_equal(nbr_g, nbr_o)
    gl_o = o.ghost_list()
    gl_g = g.ghost_list()
    assert gl_g.shape == gl_o.shape == (g.n_blocks * 1216, 9)
    assert np.array_equal(gl_g, gl_o)
    # the per-cell plan the product kernel reads decodes to the same tuples
    assert np.array_equal(g.ghost_list(from_plan=True), gl_o)
    g.close()


def test_plan_patterns_are_shared():
    # blocks with identical surroundings share one plan pattern: a uniform periodic grid
    # with >= 3 blocks per axis has exactly one; the AMR grid of config 3 has a handful
    import paper_2501_06717_b200 as batl
    g = batl.Grid(wl.random_uniform((4, 3, 3)))
    assert g.plan_patterns().shape == (1, 1216)
    g.close()
    g = batl.Grid(wl.brio_wu_amr())
    n = g.plan_patterns().shape[0]
    assert 1 < n < g.n_blocks // 4
    g.close()


def test_message_sizes_match_paper_L146():
    # PAPER.md L146 scaled to 8^3 blocks: face 128 cells, edge 32, corner 8;
    # towards a coarser... from a finer neighbour the face splits into 4 messages of 4x4x2
    import paper_2501_06717_b200 as batl
    g = batl.Grid(wl.random_uniform((2, 2, 2)))
    m = g.ghost_messages()
    assert len(m) == 8 * 26
    cells = m["n"].astype(int).prod(axis=1)
    nd = np.array([sum(1 for q in (d % 3, (d // 3) % 3, d // 9) if q != 1) for d in m["dir"]])
    assert set(cells[nd == 1]) == {128} and set(cells[nd == 2]) == {32} and set(cells[nd == 3]) == {8}
    assert (m["kind"] == 0).all()
    g.close()
    g = batl.Grid(wl.fast_wave((2, 2, 2)))
    m = g.ghost_messages()
    r = m[m["kind"] == 1]
    cells = r["n"].astype(int).prod(axis=1)
    nd = np.array([sum(1 for q in (d % 3, (d // 3) % 3, d // 9) if q != 1) for d in r["dir"]])
    assert set(cells[nd == 1]) == {32} and set(cells[nd == 2]) == {16} and set(cells[nd == 3]) == {8}
    g.close()


def test_invalid_configs_are_rejected():
    import paper_2501_06717_b200 as batl
    bad = dict(wl.alfven())
    bad["bc"] = (0, 1, 0, 0, 0, 0)           # periodic must pair
    with pytest.raises(batl.BatlError):
        batl.Grid(bad)
    bad = dict(wl.alfven())
    bad["gamma"] = 1.0
    with pytest.raises(batl.BatlError):
        batl.Grid(bad)
    bad = dict(wl.alfven())
    bad["dt_mode"], bad["dt_fixed"] = wl.DT_FIXED, 0.0
    with pytest.raises(batl.BatlError):
        batl.Grid(bad)


def test_no_cpu_fallback_without_device():
    # the product path must fail loudly when there is no GPU
    import torch
    import paper_2501_06717_b200 as batl
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    g = batl.Grid(wl.alfven())
    with pytest.raises(batl.BatlError):
        g.bind()
    with pytest.raises(batl.BatlError):
        g.step(1)
    g.close()


# ---- host tables of the resolution-change operators -------------------------------
def _three_level_cfg():
    cfg = dict(wl.fast_wave((2, 2, 2)))
    cfg["regions"] = [(wl.SHAPE_BOX, 1, (-32.0, -32.0, -32.0, 0.0, 0.0, 0.0)),
                      (wl.SHAPE_SPHERE, 3, (-30.0, -30.0, -30.0, 3.0, 0.0, 0.0))]
    cfg["max_level"] = 3
    cfg["bc"] = (wl.BC_FLOAT, wl.BC_FLOAT, wl.BC_PERIODIC, wl.BC_PERIODIC, wl.BC_FLOAT, wl.BC_FLOAT)
    return cfg


@pytest.mark.parametrize("make", [lambda: wl.fast_wave((2, 2, 2)), _three_level_cfg, _mixed_bc_amr, wl.brio_wu_amr])
def test_second_order_prolongation_plan_child_parities(make):
    # Q-G4b: a plan entry of kind PLAN_PROLONG2 carries, per axis, whether the fine ghost cell is the high
    # child of its coarse source cell = the parity of its global fine coordinate after the periodic wrap or
    # the clamp at a float boundary.  Recomputed here from the geometry alone.
    import paper_2501_06717_b200 as batl
    cfg = dict(make(), prolong_order=2)
    g = batl.Grid(cfg)
    blocks = g.blocks()
    pats, ids = g.plan_patterns(), g.plan_ids()
    n_checked = 0
    for b, (lev, I, J, K) in enumerate(blocks):
        for e in pats[ids[b]]:
            kind = int(e) >> 28
            if kind < 8:
                continue
            sd = int(e) & 2047
            c = (sd % 12 - 2, (sd // 12) % 12 - 2, sd // 144 - 2)
            for a, (root, ca, Ia) in enumerate(zip(cfg["n_root"], c, (I, J, K))):
                N = (8 * root) << lev
                gco = 8 * Ia + ca
                if gco < 0 or gco >= N:
                    face = 2 * a + (1 if gco >= N else 0)
                    if cfg["bc"][face] == wl.BC_PERIODIC:
                        gco %= N
                    else:
                        gco = 0 if gco < 0 else N - 1
                assert (kind >> a) & 1 == gco & 1, (b, c, a)
            n_checked += 1
    assert n_checked > 0
    # first order: no such entries
    assert not (batl.Grid(make()).plan_patterns() >> 28 >= 8).any()


@pytest.mark.parametrize("make", [lambda: wl.fast_wave((2, 2, 2)), _three_level_cfg, wl.magnetosphere])
def test_flux_correction_tables_follow_the_neighbour_table(make):
    # Q-G6b: a slot for every block face at a resolution change (both sides), none elsewhere; one record per
    # face that borders finer blocks, naming the slots of those four blocks' opposite faces in the order of
    # the neighbour table (lower tangential axis fastest)
    import paper_2501_06717_b200 as batl
    g = batl.Grid(dict(make(), flux_correction=1))
    nbr, dlev = g.neighbors()
    slots, recs = g.flux_correction_tables()
    face_dirs = [12, 14, 10, 16, 4, 22]
    jump = np.isin(dlev[:, face_dirs], (-1, 1))
    assert np.array_equal(slots >= 0, jump)
    used = np.sort(slots[slots >= 0])
    assert np.array_equal(used, np.arange(len(used)))            # dense, each slot once
    coarse_faces = {(b, f) for b in range(g.n_blocks) for f in range(6) if dlev[b, face_dirs[f]] == -1}
    assert {(int(r[0]), int(r[1])) for r in recs} == coarse_faces and len(recs) == len(coarse_faces)
    for b, f, own, f0, f1, f2, f3, _ in recs:
        assert own == slots[b, f]
        fine = nbr[b, face_dirs[f]]
        assert [f0, f1, f2, f3] == [slots[fb, f ^ 1] for fb in fine]
        assert all(dlev[fb, face_dirs[f ^ 1]] == 1 for fb in fine)
    assert np.array_equal(np.sort(recs[:, 0]), recs[:, 0])       # grouped by block, ascending
    # switched off: no slots, no records
    s0, r0 = batl.Grid(make()).flux_correction_tables()
    assert (s0 < 0).all() and len(r0) == 0
