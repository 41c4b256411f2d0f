"""Pins of the oracle's resolution-change operators of SURVEY.md 8(f) rank 3 (PAPER.md L128 names
restriction / prolongation / copy and gives no formula; L168 calls the scheme "nearly conservative";
L185: the refined octant exists "to test our algorithm's ability to deal with a change in grid
resolution"): second-order limited prolongation (reading Q-G4b) and conservative flux correction
(reading Q-G6b).  Expected values come from the mathematics -- a linear field is reproduced
exactly, the eight children of a coarse cell average to it, totals are conserved to round-off, a
first-order closed form of the corrected coarse cell -- never from the oracle itself.
"""
import numpy as np
import pytest

import oracle
import workloads as wl

NI, NG, NS = 8, 2, 12


def _amr_cfg(**kw):
    cfg = dict(wl.fast_wave((2, 2, 2)))            # the paper's grid: 2^3 roots, one octant refined (15 leaves)
    cfg.update(kw)
    return cfg


def _three_level():
    cfg = dict(wl.fast_wave((2, 2, 2)))
    cfg["regions"] = [(wl.SHAPE_BOX, 1, (-32.0, -32.0, -32.0, 0.0, 0.0, 0.0)),
                      (wl.SHAPE_SPHERE, 3, (-30.0, -30.0, -30.0, 3.0, 0.0, 0.0))]
    cfg["max_level"] = 3
    cfg["bc"] = (wl.BC_FLOAT, wl.BC_FLOAT, wl.BC_PERIODIC, wl.BC_PERIODIC, wl.BC_FLOAT, wl.BC_FLOAT)
    return cfg


def _centres_with_ghosts(cfg, blk):
    d = wl.cell_size(cfg, blk[0])
    idx = np.arange(-NG, NI + NG) + 0.5
    return [cfg["xyz_min"][a] + (NI * int(blk[1 + a]) + idx) * d[a] for a in range(3)]


def _totals(cfg, blocks, U):
    """sum over all physical cells of U times the cell volume, per variable"""
    vol = np.array([np.prod(wl.cell_size(cfg, b[0])) for b in blocks])
    return (U.reshape(len(blocks), 8, -1).sum(axis=2) * vol[:, None]).sum(axis=0)


# --------------------------------------------------------------------------- Q-G4b
def test_second_order_prolongation_reproduces_a_linear_field_exactly():
    # cell centres are odd integers (coarse: multiples of 2 offset by 2) and the coefficients are small
    # integers, so every difference, slope and quarter slope is exact in fp64: the fine ghost cells
    # filled from a coarser block must hold the linear field at their own centres, bit for bit.
    # A wrong sign of a quarter slope, a wrong child parity, a slope taken in the wrong direction or a
    # first-order fill all fail.  Cells whose coarse stencil touches the (periodic) domain boundary,
    # where the field jumps, are left out.
    cfg = _amr_cfg(prolong_order=2)
    o = oracle.Oracle(cfg)
    blocks = o.blocks()
    coef = np.array([[3, 1, -2, 4], [5, -3, 2, 1], [-7, 2, 5, -1], [11, 4, 1, 3],
                     [2, -1, -4, 2], [-9, 3, 3, 3], [6, -5, 1, -2], [40, 2, -3, 5]], dtype=np.float64)

    def field(v, X, Y, Z):
        return coef[v, 0] + coef[v, 1] * X + coef[v, 2] * Y + coef[v, 3] * Z

    U = np.zeros((len(blocks), 8, NI, NI, NI))
    for b, blk in enumerate(blocks):
        x, y, z = wl.cell_centres(cfg, blk)
        for v in range(8):
            U[b, v] = field(v, x[None, None, :], y[None, :, None], z[:, None, None])
    o.set_state(U)
    S = o.get_state(True)
    gl = o.ghost_list()
    prolonged = gl[gl[:, 4] == 2]
    assert len(prolonged) > 0
    checked = 0
    for dst, k, j, i, _, _, _, _, _ in prolonged:
        x, y, z = _centres_with_ghosts(cfg, blocks[dst])
        p = np.array([x[i + NG], y[j + NG], z[k + NG]])
        # the coarse cell and its six neighbours (cell size 4) must stay clear of the boundary at +-32
        # (the wrap) by more than one coarse cell plus the restriction footprint
        if np.any(np.abs(p) > 32.0 - 10.0):
            continue
        for v in range(8):
            assert S[dst, v, k + NG, j + NG, i + NG] == field(v, p[0], p[1], p[2]), (dst, k, j, i, v)
        checked += 1
    assert checked > 500

    # first-order prolongation (Q-G4) holds the coarse value instead: the test has teeth
    o1 = oracle.Oracle(_amr_cfg(prolong_order=1))
    o1.set_state(U)
    assert not np.array_equal(o1.get_state(True), S)


def test_second_order_prolongation_children_average_to_the_coarse_cell():
    # the eight fine ghost cells cut from one coarse cell take +-1/4 of each slope with all sign
    # combinations: their mean is the coarse value (conservation of the prolongation operator)
    cfg = _amr_cfg(prolong_order=2)
    cfg["field"] = "random"
    o = oracle.Oracle(cfg)
    blocks = o.blocks()
    o.set_primitive(wl.initial_primitive(cfg, blocks))
    S = o.get_state(True)
    gl = o.ghost_list()
    pro = gl[gl[:, 4] == 2]
    # group the prolonged ghost cells by (destination block, source block, source cell)
    groups = {}
    for dst, k, j, i, _, src, ks, js, is_ in pro:
        groups.setdefault((dst, src, ks, js, is_), []).append((k, j, i))
    n = 0
    for (dst, src, ks, js, is_), cells in groups.items():
        if len(cells) != 8:
            continue                         # clipped at an edge of the ghost layer
        for v in range(8):
            vals = [S[dst, v, k + NG, j + NG, i + NG] for k, j, i in cells]
            c0 = S[src, v, ks + NG, js + NG, is_ + NG]
            assert abs(np.mean(vals) - c0) <= 4e-16 * max(1.0, abs(c0))
        n += 1
    assert n > 100


def test_second_order_prolongation_is_bounded_by_the_coarse_neighbours_in_1d():
    # data that vary along x only: the prolonged value is U_C +- s/4 with |s| <= 2 min|D|, so it lies
    # between U_C and the coarse neighbour on that side (no new extrema), and equals U_C at an extremum
    cfg = _amr_cfg(prolong_order=2)
    o = oracle.Oracle(cfg)
    blocks = o.blocks()
    rng = np.random.default_rng(7)
    prof = {}                                # value per distinct x of the coarse level (cell size 4)

    def val(xc):
        key = float(np.floor((xc + 32.0) / 4.0))
        if key not in prof:
            prof[key] = rng.uniform(1.0, 2.0)
        return prof[key]

    U = np.zeros((len(blocks), 8, NI, NI, NI))
    for b, blk in enumerate(blocks):
        x, _, _ = wl.cell_centres(cfg, blk)
        row = np.array([val(xx) for xx in x])          # fine cells inherit the value of their coarse column
        U[b, :] = row[None, None, None, :]
    o.set_state(U)
    S = o.get_state(True)
    gl = o.ghost_list()
    n = 0
    for dst, k, j, i, kind, src, ks, js, is_ in gl[gl[:, 4] == 2]:
        c0 = S[src, 0, ks + NG, js + NG, is_ + NG]
        lo = S[src, 0, ks + NG, js + NG, is_ - 1 + NG]
        hi = S[src, 0, ks + NG, js + NG, is_ + 1 + NG]
        got = S[dst, 0, k + NG, j + NG, i + NG]
        assert min(lo, c0, hi) - 1e-15 <= got <= max(lo, c0, hi) + 1e-15
        if (c0 - lo) * (hi - c0) <= 0.0:
            assert got == c0                           # extremum: zero slope, first-order value
        n += 1
    assert n > 1000


@pytest.mark.parametrize("make", [_amr_cfg, _three_level, wl.brio_wu_amr, wl.magnetosphere])
def test_second_pass_of_the_prolongation_reads_no_prolonged_cell(make):
    # the two-pass order (copy / restriction / boundary states first, prolongation second) is only
    # well defined if the coarse stencil never contains a prolonged ghost cell: true under the
    # nesting rule Q-O2 (level jumps <= 1 across faces, edges and corners)
    assert oracle.Oracle(make()).prolong_reads_prolonged() == 0


def test_uniform_state_is_preserved_bit_identically_with_both_operators():
    cfg = wl.uniform_state(_three_level())
    cfg.update(prolong_order=2, flux_correction=1)
    o = oracle.Oracle(cfg)
    o.set_primitive(wl.initial_primitive(cfg, o.blocks()))
    U0 = o.get_state(True)
    o.step(5)
    assert np.array_equal(o.get_state(True), U0)


# --------------------------------------------------------------------------- Q-G6b
@pytest.mark.parametrize("prolong_order", [1, 2])
def test_flux_correction_conserves_on_the_periodic_amr_grid(prolong_order):
    # T3 on an AMR grid: with the 8-wave source off every equation is a conservation law, and with
    # the coarse face flux replaced by the mean of the fine ones the volume-weighted totals of all
    # eight variables are constant to round-off.  Without the correction they drift visibly (the
    # paper's "nearly conservative", L168): the test has teeth.
    drift = {}
    for fc in (1, 0):
        cfg = _amr_cfg(prolong_order=prolong_order, flux_correction=fc, use_divb_source=0)
        cfg["field"] = "random"
        o = oracle.Oracle(cfg)
        blocks = o.blocks()
        o.set_primitive(wl.initial_primitive(cfg, blocks))
        T0 = _totals(cfg, blocks, o.get_state())
        scale = np.array([np.abs(T0[0]), np.abs(T0[7]) ** 0.5 * np.abs(T0[0]) ** 0.5] + [1.0] * 6)   # not used for zeros
        w, _, _ = o.step(5)
        assert w == 0
        T1 = _totals(cfg, blocks, o.get_state())
        # momentum and field totals are O(1) * volume; scale everything by the total volume times the
        # typical magnitude of the variable (rho ~ 1, |rho u| ~ 0.1, |B| ~ 1, e ~ 2)
        vol = 64.0 ** 3
        mag = np.array([1.0, 0.1, 0.1, 0.1, 1.0, 1.0, 0.1, 2.0]) * vol
        drift[fc] = np.abs(T1 - T0) / mag
    assert drift[1].max() <= 1e-13, drift[1]
    assert drift[0].max() >= 1e-9, drift[0]


def test_flux_correction_closed_form_first_order_density_advection():
    # One first-order one-stage step with fixed dt of rho(x, y, z) advected by a uniform flow along x
    # (uniform u = (u, 0, 0), p; B = 0).  Every density flux is the closed-form Rusanov flux of two cell
    # values, written out here in numpy:
    #   x faces: F(a, b) = u (a + b)/2 - c(a, b) (b - a)/2,   y, z faces: G(a, b) = -c0(a, b) (b - a)/2,
    #   c = |u| + sqrt(gamma p / ((a + b)/2)),  c0 = sqrt(gamma p / ((a + b)/2)).
    # A coarse cell (j, k) right of the fine octant (across x = 0) then holds
    #   rho - dt/D (F(rho, rho_right) - F_lo) - dt/D (dG_y + dG_z),
    # with F_lo = the MEAN of the four fine fluxes F(rho_fine_last(j', k'), rho) over the fine faces
    # (j', k') = (2j + {0,1}, 2k + {0,1}) that cover the coarse face (the fine ghost is the first-order
    # prolonged coarse value), whereas the uncorrected scheme uses F(restricted ghost, rho).  rho varies
    # in y and z, so taking the fluxes of the wrong fine block or quadrant shows.
    gamma, u, p, dt = 5.0 / 3.0, 0.3, 0.8, 0.5

    def rho_of(x, y, z):
        return 1.0 + 0.3 * np.sin(0.11 * x) + 0.002 * x + 0.05 * np.sin(0.2 * y + 0.3 * z)

    results = {}
    for fc in (0, 1):
        cfg = _amr_cfg(n_stage=1, n_order=1, flux_correction=fc, dt_mode=wl.DT_FIXED, dt_fixed=dt, use_divb_source=1)
        o = oracle.Oracle(cfg)
        blocks = o.blocks()
        W = np.zeros((len(blocks), 8, NI, NI, NI))
        for b, blk in enumerate(blocks):
            x, y, z = wl.cell_centres(cfg, blk)
            W[b, 0] = rho_of(x[None, None, :], y[None, :, None], z[:, None, None])
            W[b, 1] = u
            W[b, 7] = p
        o.set_primitive(W)
        rho0 = o.get_state(True)[:, 0]
        o.step(1)
        results[fc] = (blocks, rho0, o.get_state()[:, 0])

    def c0(a, b):
        return np.sqrt(gamma * p / (0.5 * (a + b)))

    def F(a, b):
        return u * 0.5 * (a + b) - 0.5 * (abs(u) + c0(a, b)) * (b - a)

    def G(a, b):
        return -0.5 * c0(a, b) * (b - a)

    for fc in (0, 1):
        blocks, rho0, rho1 = results[fc]
        index = {tuple(blk): b for b, blk in enumerate(blocks)}
        bc = index[(0, 1, 0, 0)]                      # coarse block whose -x face borders the fine octant
        D = wl.cell_size(cfg, 0)[0]
        for j, k in ((0, 0), (5, 2), (2, 6), (7, 7)):   # the four quadrants of the face = four fine blocks
            R = rho0[bc]

            def at(i_, j_, k_):
                return R[k_ + NG, j_ + NG, i_ + NG]

            r = at(0, j, k)
            bf = index[(1, 1, j // 4, k // 4)]        # the fine block left of the face cell
            fine = [rho0[bf, 2 * (k % 4) + dk + NG, 2 * (j % 4) + dj + NG, 7 + NG] for dk in (0, 1) for dj in (0, 1)]
            if fc:
                F_lo = np.mean([F(f, r) for f in fine])
            else:
                F_lo = F(at(-1, j, k), r)             # the restricted ghost cell of the coarse block
            expect = r - dt / D * (F(r, at(1, j, k)) - F_lo) \
                       - dt / D * (G(r, at(0, j + 1, k)) - G(at(0, j - 1, k), r)) \
                       - dt / D * (G(r, at(0, j, k + 1)) - G(at(0, j, k - 1), r))
            assert abs(rho1[bc, k, j, 0] - expect) <= 4e-15, (fc, j, k, rho1[bc, k, j, 0], expect)
    # and the two schemes really differ in those cells
    assert abs(results[0][2] - results[1][2]).max() > 1e-6
