"""Parity of the CUDA path (through the C ABI) against the CPU oracle on the same
seeded inputs.  Bar (BASELINE.json north_star): ghost values bit-identical, state
within 1e-11 max relative error (norm O-9 of DESIGN.md) after the steps."""
import os

import numpy as np
import pytest

import workloads as wl
from util import rel_err_O9, rel_err_per_block

pytestmark = pytest.mark.gpu

TOL = 1e-11          # north_star: max relative error on all state variables (fp64)


def _mixed_bc_amr():
    cfg = dict(wl.fast_wave((2, 2, 2)))
    cfg["bc"] = (wl.BC_FLOAT, wl.BC_FIXED, wl.BC_FLOAT, wl.BC_FLOAT, wl.BC_PERIODIC, wl.BC_PERIODIC)
    bp = np.zeros((6, 8))
    bp[1] = (1.05, 0.004, 0.0, 0.0, 0.0, 0.0404, 0.0, 0.00058)
    cfg["bc_prim"] = bp
    return cfg


def _three_level():
    cfg = dict(wl.fast_wave((2, 2, 2)))
    cfg["regions"] = [(wl.SHAPE_BOX, 1, (-32.0, -32.0, -32.0, 0.0, 0.0, 0.0)),
                      (wl.SHAPE_SPHERE, 3, (-30.0, -30.0, -30.0, 3.0, 0.0, 0.0))]
    cfg["max_level"] = 3
    cfg["bc"] = (wl.BC_FLOAT, wl.BC_FLOAT, wl.BC_PERIODIC, wl.BC_PERIODIC, wl.BC_FLOAT, wl.BC_FLOAT)
    return cfg


def _pair(orc, cfg, variant=0, perturb=False):
    """Oracle and bound GPU grid holding the same initial conserved state."""
    import paper_2501_06717_b200 as batl
    o = orc.Oracle(cfg)
    g = batl.Grid(cfg).bind()
    g.set_kernel_variant(variant)
    blocks = o.blocks()
    assert np.array_equal(g.blocks(), blocks)
    W = wl.initial_primitive(cfg, blocks)
    if perturb:      # make every cell distinct so that index slips cannot hide
        rng = np.random.default_rng(cfg["seed"] + 77)
        W[:, 0] *= 1.0 + 0.01 * rng.uniform(-1, 1, size=W[:, 0].shape)
        W[:, 7] *= 1.0 + 0.01 * rng.uniform(-1, 1, size=W[:, 7].shape)
        W[:, 1:7] += 1e-3 * np.abs(W[:, 1:7]).max() * rng.uniform(-1, 1, size=W[:, 1:7].shape)
    o.set_primitive(W)
    U0 = o.get_state()
    g.set_state(U0)
    return o, g


GHOST_CASES = {
    # second-order limited prolongation (Q-G4b, two-pass fill): same bar, every ghost value bit-identical
    "fast_wave_15_prolong2": lambda: dict(wl.fast_wave((2, 2, 2)), prolong_order=2),
    "brio_wu_amr_prolong2": lambda: dict(wl.brio_wu_amr(), prolong_order=2),
    "mixed_bc_amr_prolong2": lambda: dict(_mixed_bc_amr(), prolong_order=2),
    "three_level_prolong2": lambda: dict(_three_level(), prolong_order=2),
    "alfven": lambda: wl.alfven(),
    "uniform_1x1x1": lambda: wl.random_uniform((1, 1, 1)),
    "uniform_2x1x3": lambda: wl.random_uniform((2, 1, 3)),
    "fast_wave_15": lambda: wl.fast_wave((2, 2, 2)),
    "brio_wu_amr": lambda: wl.brio_wu_amr(),
    "mixed_bc_amr": _mixed_bc_amr,
    "three_level": _three_level,
}


@pytest.mark.parametrize("name", sorted(GHOST_CASES))
def test_ghost_fill_bit_identical(orc, name):
    cfg = GHOST_CASES[name]()
    o, g = _pair(orc, cfg, perturb=True)
    ref = o.get_state(with_ghost=True)
    got = g.get_state(with_ghost=True)
    assert np.array_equal(got, ref), f"{(got != ref).sum()} ghost/physical values differ"
    g.close()


def _run_and_compare(orc, cfg, n_steps, variant=0, check_dt=True):
    o, g = _pair(orc, cfg, variant=variant)
    wo, to, dto = o.step(n_steps)
    wg, tg, dtg = g.step(n_steps)
    ref = o.get_state(with_ghost=True)
    got = g.get_state(with_ghost=True)
    err = rel_err_O9(got, ref)
    assert np.isfinite(got).all()
    assert err <= TOL, f"relative error {err:.3e} > {TOL}"
    assert wg == wo
    if check_dt and cfg["dt_mode"] != wl.DT_LOCAL:
        assert abs(tg - to) <= 1e-12 * abs(to)
        assert abs(dtg - dto) <= 1e-12 * abs(dto)
    g.close()
    return err


@pytest.mark.parametrize("variant", [0, 1])
def test_config1_alfven_10_steps(orc, variant):
    # BASELINE.json configs[0]: 2x2x2 blocks, Alfven wave, CFL 0.8, 10 steps
    _run_and_compare(orc, wl.alfven(), 10, variant)


@pytest.mark.parametrize("variant", [0, 1])
def test_config2_orszag_tang_10_steps(orc, variant):
    # configs[1] at full size (512 blocks); 10 steps (north_star: error after 10 steps)
    _run_and_compare(orc, wl.orszag_tang(), 10, variant)


@pytest.mark.parametrize("variant", [0, 1])
def test_config3_brio_wu_amr_10_steps(orc, variant):
    # configs[2]: two-level AMR, float x boundaries, shock
    _run_and_compare(orc, wl.brio_wu_amr(), 10, variant)


@pytest.mark.parametrize("variant", [0, 1])
def test_config4_random_ragged_grid(orc, variant):
    # configs[3] recipe on a grid whose block count (5*3*2 = 30) is not a multiple of anything convenient
    _run_and_compare(orc, wl.random_uniform((5, 3, 2)), 10, variant)


def test_config4_full_size_4096_blocks(orc):
    # the bench configuration (16^3 blocks) in the launch configuration bench.py times, for the
    # north_star's 10 steps
    _run_and_compare(orc, wl.random_uniform((16, 16, 16)), 10)


def test_config4_full_length_50_steps(orc):
    # BASELINE.json configs[3] at its own step count (50) and size (4,096 blocks)
    _run_and_compare(orc, wl.random_uniform((16, 16, 16)), 50)


def test_config4_sweep_points_below_and_above_the_bench_point(orc):
    # the throughput sweep of configs[3] against the oracle on both sides of 4,096 blocks
    _run_and_compare(orc, wl.random_uniform((16, 16, 8)), 3)       # 2,048 blocks
    _run_and_compare(orc, wl.random_uniform((32, 16, 16)), 2)      # 8,192 blocks


def test_config5_magnetosphere_3_steps(orc):
    # configs[4]: 4 levels, B0 dipole, body, fixed inflow, float outflow, local dt
    cfg = wl.magnetosphere()
    o, g = _pair(orc, cfg)
    wo, _, _ = o.step(3)
    wg, _, _ = g.step(3)
    ref, got = o.get_state(True), g.get_state(True)
    assert rel_err_O9(got, ref) <= TOL
    # four refinement levels and a solar-wind / near-body contrast: also block by block
    per_block = rel_err_per_block(g.get_state(), o.get_state())
    print("config 5, 3 steps, per-block relative error:", per_block)
    assert max(per_block.values()) <= TOL, per_block
    dto, dtg = o.get_dt_local(), g.get_dt_local()
    assert np.abs(dtg - dto).max() <= 1e-12 * np.abs(dto).max()
    assert wg == wo
    # the blocks with body cells run in the fused kernel too (BODY variant): no general-kernel launch
    kc = g.kernel_counts()
    assert kc["general"] == 0 and kc["fused"] > 0, kc
    g.close()


@pytest.mark.parametrize("variant", [0, 1])
def test_fast_wave_amr_fixed_dt(orc, variant):
    # paper's fast-wave set-up on the 15-leaf grid (L185, L339-343), fixed dt so that
    # the result does not depend on the dt reduction
    cfg = dict(wl.fast_wave((2, 2, 2)))
    cfg["dt_mode"], cfg["dt_fixed"] = wl.DT_FIXED, 2.0
    _run_and_compare(orc, cfg, 10, variant)


@pytest.mark.parametrize("variant", [0, 1])
def test_mixed_bc_three_level(orc, variant):
    _run_and_compare(orc, _three_level(), 5, variant)
    _run_and_compare(orc, _mixed_bc_amr(), 5, variant)


def test_local_dt_uniform_grid(orc):
    cfg = wl.random_uniform((2, 2, 2), dt_mode=wl.DT_LOCAL)
    _run_and_compare(orc, cfg, 5)


def test_uniform_b0_split_on_gpu(orc):
    # use_b0 = 2 (uniform B0): exercises every B0 term of flux and source on the GPU
    cfg = wl.random_uniform((2, 2, 2), use_b0=2, dipole_m=(0.3, -0.2, 0.5))
    _run_and_compare(orc, cfg, 5)


def test_other_limiter_beta_and_flux_fallbacks(orc):
    # beta = 1.5: the fused kernel without the beta = 2 special case
    _run_and_compare(orc, wl.random_uniform((3, 2, 2), limiter_beta=1.5), 5)
    # HLL flux with a uniform B0 and global dt has no fused variant: general kernel on every block,
    # and batl_kernel_counts says so
    import paper_2501_06717_b200 as batl
    cfg = wl.random_uniform((2, 2, 2), use_b0=2, dipole_m=(0.3, -0.2, 0.5), flux_type=1)
    _run_and_compare(orc, cfg, 4)
    g = batl.Grid(cfg).bind()
    g.set_state(wl.initial_conserved(cfg, g.blocks()))
    g.step(1)
    assert g.kernel_counts()["general_fallback"] == 3 and g.kernel_counts()["fused"] == 0
    g.close()
    # local dt without B0 (fused LDT variant), first order with B0 but global dt (beta = 0 path)
    _run_and_compare(orc, wl.random_uniform((2, 2, 2), dt_mode=wl.DT_LOCAL), 4)
    _run_and_compare(orc, wl.random_uniform((2, 2, 2), use_b0=2, dipole_m=(0.3, -0.2, 0.5), n_order=1, n_stage=1, cfl=0.4), 4)


def test_no_divb_source(orc):
    _run_and_compare(orc, wl.random_uniform((2, 2, 2), use_divb_source=0), 5)


def test_uniform_state_is_preserved_bit_identically(orc):
    # degenerate case: constant state on the AMR grid stays constant to the last bit
    cfg = wl.uniform_state(wl.fast_wave((2, 2, 2)))
    o, g = _pair(orc, cfg)
    U0 = g.get_state(True)
    g.step(5)
    assert np.array_equal(g.get_state(True), U0)
    g.close()


def test_step_splitting_and_determinism(orc):
    # mhd_step(4) == 4 x mhd_step(1), bit for bit, and two runs agree bit for bit
    cfg = wl.random_uniform((3, 2, 2))
    _, g1 = _pair(orc, cfg)
    _, g2 = _pair(orc, cfg)
    g1.step(4)
    for _ in range(4):
        g2.step(1)
    assert np.array_equal(g1.get_state(True), g2.get_state(True))
    g1.close()
    g2.close()


def test_persistent_pipeline_is_race_free_at_bench_scale():
    # 2,048 blocks = 4,096 half blocks over 296 persistent CTAs: every CTA pipelines ~14 tiles
    # (TMA prefetch into a tile it has just stopped reading, exchange buffers reused across
    # iterations without a closing barrier).  A race would make repeated runs differ; they must
    # agree bit for bit, and the fused kernel must agree with the general kernel to round-off.
    import paper_2501_06717_b200 as batl
    # second case: an AMR grid, where consecutive half blocks of a CTA differ in cell
    # size, so that a per-tile scalar published too early would show (960 blocks, ~6 tiles per CTA;
    # compute-sanitizer is closed on this pool, profiles/r02_sanitizer.md)
    for cfg in (wl.random_uniform((16, 16, 8)), wl.fast_wave((8, 8, 8))):
        g = batl.Grid(cfg).bind()
        U0 = wl.initial_conserved(cfg, g.blocks())
        runs = []
        for variant in (0, 0, 0, 1):
            g.set_kernel_variant(variant)
            g.set_state(U0)
            g.step(3)
            runs.append(g.get_state(True))
        assert np.array_equal(runs[0], runs[1]) and np.array_equal(runs[0], runs[2])
        assert rel_err_O9(runs[0], runs[3]) <= 1e-12
        g.close()


@pytest.mark.parametrize("name,n_steps", [("orszag_tang", 100), ("brio_wu_amr", 200), ("magnetosphere", 100)])
def test_full_length_runs_of_configs_2_3_5(orc, name, n_steps):
    # BASELINE.json's step counts, not just 10 steps: the error stays at round-off level
    cfg = getattr(wl, name)()
    o, g = _pair(orc, cfg)
    wo, _, _ = o.step(n_steps)
    wg, _, _ = g.step(n_steps)
    assert rel_err_O9(g.get_state(True), o.get_state(True)) <= TOL
    per_block = rel_err_per_block(g.get_state(), o.get_state())
    print(name, n_steps, "steps, per-block relative error:", per_block)
    assert max(per_block.values()) <= TOL, per_block
    assert wg == wo == 0
    g.close()


def test_largest_sweep_point_properties():
    # 32^3 = 32,768 blocks (16.8 M cells, 2 x 3.6 GB of state): the top of config 4's sweep, too big
    # for the oracle, so checked through what holds at any size: a uniform state is a fixed point
    # bit for bit, mass is conserved to round-off on the periodic grid, ghost cells equal the
    # physical cells they copy (periodic wrap included) bit for bit, and no warning is raised
    import paper_2501_06717_b200 as batl
    cfg = wl.random_uniform((32, 32, 32))
    g = batl.Grid(cfg).bind()
    nB = g.n_blocks
    assert nB == 32768
    rng = np.random.default_rng(5)
    U = np.empty((nB, 8, 8, 8, 8))
    U[:, 0] = 1.0 + 0.05 * rng.standard_normal((nB, 8, 8, 8)).clip(-4, 4)
    U[:, 1:4] = 0.1 * rng.standard_normal((nB, 3, 8, 8, 8)).clip(-4, 4)
    U[:, 4:7] = np.array([0.7, 0.7, 0.0])[None, :, None, None, None] + 0.1 * rng.standard_normal((nB, 3, 8, 8, 8)).clip(-4, 4)
    U[:, 7] = 2.5 + 0.1 * rng.standard_normal((nB, 8, 8, 8)).clip(-4, 4)
    g.set_state(U)
    m0 = U[:, 0].sum()
    w, t, dt = g.step(2)
    assert w == 0 and t > 0
    V = g.get_state(True)
    assert np.isfinite(V).all()
    assert abs(V[:, 0, 2:10, 2:10, 2:10].sum() - m0) <= 1e-12 * m0
    blk = g.blocks()
    idx = {(int(i), int(j), int(k)): b for b, (_, i, j, k) in enumerate(blk)}
    for b in (0, 1, 31, 1023, 17000, nB - 1):                 # x faces of a few blocks, wrap included
        _, i, j, k = (int(q) for q in blk[b])
        right = idx[((i + 1) % 32, j, k)]
        left = idx[((i - 1) % 32, j, k)]
        assert np.array_equal(V[b, :, 2:10, 2:10, 10:12], V[right, :, 2:10, 2:10, 2:4])
        assert np.array_equal(V[b, :, 2:10, 2:10, 0:2], V[left, :, 2:10, 2:10, 8:10])
    del V
    U[:] = np.array([1.3, 0.26, -0.13, 0.065, 0.7, -0.4, 0.3, 2.0])[None, :, None, None, None]
    g.set_state(U)
    g.step(2)
    assert np.array_equal(g.get_state(), U)
    g.close()


def test_body_blocks_split_between_the_two_kernels(orc):
    # body without B0 and with global dt: fused kernel on the block list + general kernel on the body blocks
    cfg = dict(wl.magnetosphere())
    cfg["use_b0"], cfg["dt_mode"] = 0, wl.DT_GLOBAL
    cfg["regions"] = cfg["regions"][:2]
    cfg["max_level"] = 2
    _run_and_compare(orc, cfg, 2)


@pytest.mark.parametrize("variant", [0, 1])
@pytest.mark.parametrize("n_order", [1, 2])
def test_one_stage_scheme_uniform_and_amr(orc, variant, n_order):
    # Q-U2: U^{n+1} = U^n + dt R(U^n); n_order 1 = piecewise-constant states
    cfg = dict(wl.random_uniform((3, 2, 2)))
    cfg.update(n_stage=1, n_order=n_order, cfl=0.4)
    _run_and_compare(orc, cfg, 7, variant)                  # odd step count: buffers end up swapped
    cfg = dict(wl.fast_wave((2, 2, 2)))
    cfg.update(n_stage=1, n_order=n_order, cfl=0.4)
    _run_and_compare(orc, cfg, 4, variant)


def test_one_stage_magnetosphere_local_dt(orc):
    # the paper's operational setting (1-stage, first order, CFL 0.85) on config 5's grid and physics
    cfg = dict(wl.magnetosphere())
    cfg.update(n_stage=1, n_order=1, cfl=0.85)
    o, g = _pair(orc, cfg)
    wo, _, _ = o.step(3)
    wg, _, _ = g.step(3)
    assert rel_err_O9(g.get_state(True), o.get_state(True)) <= TOL
    dto, dtg = o.get_dt_local(), g.get_dt_local()
    assert np.abs(dtg - dto).max() <= 1e-12 * np.abs(dto).max()
    assert wg == wo
    g.close()


@pytest.mark.parametrize("variant", [0, 1])
def test_hll_flux_uniform_amr_and_shock(orc, variant):
    # Q-F4: the HLL-type "Linde" flux of the paper's fast-wave test (L343)
    for cfg, n in ((wl.random_uniform((3, 2, 2)), 6), (wl.fast_wave((2, 2, 2)), 6), (wl.brio_wu_amr(), 4)):
        cfg = dict(cfg)
        cfg["flux_type"] = 1
        _run_and_compare(orc, cfg, n, variant)


def test_hll_flux_magnetosphere(orc):
    cfg = dict(wl.magnetosphere())
    cfg["flux_type"] = 1
    o, g = _pair(orc, cfg)
    wo, _, _ = o.step(2)
    wg, _, _ = g.step(2)
    assert rel_err_O9(g.get_state(True), o.get_state(True)) <= TOL
    assert wg == wo
    g.close()


def test_warning_flags_match_oracle(orc):
    cfg = wl.random_uniform((2, 1, 1))
    o, g = _pair(orc, cfg)
    U = o.get_state()
    U[1, 7, 3, 3, 3] = -5.0           # negative energy -> negative pressure
    o.set_state(U)
    g.set_state(U)
    wo, _, _ = o.step(1)
    wg, _, _ = g.step(1)
    assert wo & 2 and wg & 2
    g.close()


def test_zero_steps_and_launch_count(orc):
    _, g = _pair(orc, wl.alfven())
    n0 = g.launch_count()
    w, t, dt = g.step(0)
    assert (w, t) == (0, 0.0) and g.launch_count() == n0
    g.step(2)
    # first step: stage 0 + tick; then stage 1, stage 2, tick per step -- on a uniform periodic grid the
    # stage kernels write every face ghost themselves and no ghost-fill kernel runs
    assert g.launch_count() == n0 + 2 + 2 * 3
    kc = g.kernel_counts()
    assert kc["fill_list"] == 0 and kc["general"] == 0 and kc["general_fallback"] == 0 and kc["fused"] == 1 + 2 * 2
    g.close()
    # AMR grid: only the blocks with a face at a resolution change or a boundary are filled
    _, g = _pair(orc, wl.brio_wu_amr())
    n0, f0 = g.launch_count(), g.kernel_counts()["fill_launches"]
    g.step(2)
    kc = g.kernel_counts()
    assert g.launch_count() == n0 + 2 + 2 * 5
    assert 0 < kc["fill_list"] < g.n_blocks and kc["fill_blocks"] - g.n_blocks == 4 * kc["fill_list"]
    assert kc["fill_launches"] == f0 + 4
    g.close()


PUSH_CASES = {
    "alfven": (lambda: wl.alfven(), 3),
    "uniform_1x1x1": (lambda: wl.random_uniform((1, 1, 1)), 3),         # the block is its own neighbour six times
    "uniform_2x1x3": (lambda: wl.random_uniform((2, 1, 3)), 3),
    "uniform_5x3x2": (lambda: wl.random_uniform((5, 3, 2)), 2),
    "brio_wu_amr": (lambda: wl.brio_wu_amr(), 3),
    "three_level": (_three_level, 2),
    "mixed_bc_amr": (_mixed_bc_amr, 2),
    "one_stage": (lambda: dict(wl.random_uniform((3, 2, 2)), n_stage=1, n_order=1, cfl=0.4), 3),
    "magnetosphere": (lambda: wl.magnetosphere(), 1),                       # block lists, body blocks on the general kernel
}


@pytest.mark.parametrize("name", sorted(PUSH_CASES))
def test_pushed_face_ghosts_equal_a_full_fill_bit_for_bit(orc, name):
    # row f2: after a step the FACE ghosts the next stage kernel reads (written by the neighbours' stage
    # kernels, or by the fill kernel on the fill list) are exactly what the full plan-driven fill gives;
    # edge and corner ghosts, which the scheme never reads, are only brought up to date on request
    make, n = PUSH_CASES[name]
    cfg = make()
    o, g = _pair(orc, cfg)
    g.step(n)
    raw = g.get_state(with_ghost=2)
    full = g.get_state(with_ghost=True)
    P = slice(2, 10)
    for sl in ((P, P, slice(0, 2)), (P, P, slice(10, 12)), (P, slice(0, 2), P), (P, slice(10, 12), P),
               (slice(0, 2), P, P), (slice(10, 12), P, P), (P, P, P)):
        assert np.array_equal(raw[(slice(None), slice(None)) + sl], full[(slice(None), slice(None)) + sl]), sl
    o.step(n)
    assert rel_err_O9(full, o.get_state(True)) <= TOL
    g.close()


# ---- SURVEY 8(f) rank 3, the rest: second-order prolongation (Q-G4b) and flux correction (Q-G6b) ----
AMR_OPS = [dict(prolong_order=2), dict(flux_correction=1), dict(prolong_order=2, flux_correction=1)]


@pytest.mark.parametrize("variant", [0, 1])
@pytest.mark.parametrize("ops", AMR_OPS, ids=["prolong2", "fluxcorr", "both"])
def test_resolution_change_operators_small_grids(orc, ops, variant):
    # 15-leaf periodic grid (global dt), 3-level grid with float boundaries, mixed boundary conditions
    _run_and_compare(orc, dict(wl.fast_wave((2, 2, 2), amplitude_scale=5.0), **ops), 10, variant)
    _run_and_compare(orc, dict(_three_level(), **ops), 5, variant)
    _run_and_compare(orc, dict(_mixed_bc_amr(), **ops), 5, variant)


@pytest.mark.parametrize("ops", AMR_OPS, ids=["prolong2", "fluxcorr", "both"])
def test_resolution_change_operators_config3_and_config5(orc, ops):
    # configs[2] (Brio-Wu, 352 blocks, float x boundaries) for 10 steps; configs[4] (4 levels, B0 dipole,
    # body, local dt) for 3 steps, where the correction uses the per-cell time step
    _run_and_compare(orc, dict(wl.brio_wu_amr(), **ops), 10)
    cfg = dict(wl.magnetosphere(), **ops)
    o, g = _pair(orc, cfg)
    wo, _, _ = o.step(3)
    wg, _, _ = g.step(3)
    assert rel_err_O9(g.get_state(True), o.get_state(True)) <= TOL
    assert wg == wo
    g.close()


def test_resolution_change_operators_other_schemes(orc):
    both = dict(prolong_order=2, flux_correction=1)
    # one-stage scheme, first-order face states, HLL-type flux, local dt on the 15-leaf grid
    _run_and_compare(orc, dict(wl.fast_wave((2, 2, 2)), n_stage=1, n_order=1, cfl=0.4, **both), 6)
    _run_and_compare(orc, dict(wl.fast_wave((2, 2, 2)), n_stage=1, **both), 6)
    _run_and_compare(orc, dict(wl.fast_wave((2, 2, 2)), flux_type=1, **both), 6)
    _run_and_compare(orc, dict(wl.fast_wave((2, 2, 2)), dt_mode=wl.DT_LOCAL, **both), 6)


def test_flux_correction_conserves_on_the_gpu(orc):
    # the property the operator exists for, on the device: volume-weighted totals of all eight variables
    # constant to round-off on the periodic 15-leaf grid (8-wave source off); without it they drift
    import paper_2501_06717_b200 as batl
    drift = {}
    for fc in (1, 0):
        cfg = dict(wl.fast_wave((2, 2, 2)), flux_correction=fc, use_divb_source=0, field="random")
        g = batl.Grid(cfg).bind()
        blocks = g.blocks()
        g.set_state(wl.initial_conserved(cfg, blocks))
        vol = np.array([np.prod(wl.cell_size(cfg, b[0])) for b in blocks])

        def totals():
            return (g.get_state().reshape(len(blocks), 8, -1).sum(axis=2) * vol[:, None]).sum(axis=0)

        T0 = totals()
        g.step(5)
        mag = np.array([1.0, 0.1, 0.1, 0.1, 1.0, 1.0, 0.1, 2.0]) * 64.0 ** 3
        drift[fc] = (np.abs(totals() - T0) / mag).max()
        g.close()
    assert drift[1] <= 1e-13 and drift[0] >= 1e-9, drift


def test_uniform_state_is_preserved_with_the_resolution_change_operators(orc):
    cfg = wl.uniform_state(dict(_three_level(), prolong_order=2, flux_correction=1))
    o, g = _pair(orc, cfg)
    U0 = g.get_state(True)
    g.step(5)
    assert np.array_equal(g.get_state(True), U0)
    g.close()
