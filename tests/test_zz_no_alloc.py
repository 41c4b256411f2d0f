"""mhd_stable_dt_static (include/batl.h): the CFL time step of a tiled state from an entry point that allocates
nothing -- its working data (geometry table, running minimum, warning bits) sit in a fixed device array of the
library instead of the caller-owned scratch buffer of batl_bind.  Checked against the existing path: the dt a
bound grid computes for its first step from the same state (Alg. 1 L29-64 "calculate time step";
readings Q-T1 / Q-T2 of DESIGN.md).

Collected last on purpose (the suite runs with pytest -x: a failure here hides nothing)."""
import numpy as np
import pytest

import workloads as wl

TOL = 1e-11          # the tolerance of the parity tests (tests/test_gpu_parity.py)


def test_sizes_beyond_the_static_array_are_refused_with_a_clear_error():
    # argument checks come before any CUDA call: runs without a GPU, dummy non-null pointers are never touched
    import paper_2501_06717_b200 as batl
    L = batl.lib()
    n = batl.STATIC_MAX_BLOCKS + 1
    rc = L.mhd_stable_dt_static(8, 8, n, 5.0 / 3.0, 0.8, 2.0, 2, 0, 1, 8, None, None)
    assert rc == -2                                             # BATL_ENOMEM
    msg = L.batl_static_last_error().decode()
    assert str(n) in msg and str(batl.STATIC_MAX_BLOCKS) in msg and "exceeds" in msg
    header = open(batl._build._ROOT + "/include/batl.h").read()
    assert f"#define BATL_STATIC_MAX_BLOCKS {batl.STATIC_MAX_BLOCKS}" in header
    assert L.mhd_stable_dt_static(None, 8, 1, 5.0 / 3.0, 0.8, 2.0, 2, 0, 1, 8, None, None) == -1     # null input
    assert L.mhd_stable_dt_static(8, 8, 0, 5.0 / 3.0, 0.8, 2.0, 2, 0, 1, 8, None, None) == -1        # empty


def _bound(cfg, variant):
    """A bound grid holding the configuration's initial state, its tiles (device address of block 0, variable 0:
    16 bytes into state buffer A, include/batl.h) and the per-block cell sizes on the device."""
    import torch
    import paper_2501_06717_b200 as batl
    g = batl.Grid(cfg).bind()
    g.set_kernel_variant(variant)
    blocks = g.blocks()
    g.set_state(wl.initial_conserved(cfg, blocks))              # fills every ghost cell of buffer A
    D = np.stack([wl.cell_size(cfg, b[0]) for b in blocks])
    return g, g.state_pointers()[0] + 16, torch.tensor(D, dtype=torch.float64, device="cuda:0")


@pytest.mark.gpu
def test_static_entry_point_matches_the_grid_path_on_calls_in_a_row():
    import torch
    import paper_2501_06717_b200 as batl
    # two states whose time steps differ by orders of magnitude, the second one LARGER: a running minimum
    # left over from the first call (the array keeps the last call's contents) would show up in the second;
    # the second grid is two-level, so its geometry rows differ from block to block and from the first call's
    cfg_a = wl.random_uniform((4, 4, 4))                         # 64 blocks, cell size 1/8
    cfg_b = wl.fast_wave((2, 2, 2))                              # 15 blocks, cell sizes 4 and 2
    cases = []
    for cfg in (cfg_a, cfg_b):
        g, tiles, D = _bound(cfg, 0)                             # existing path: the fused stage kernel
        g1, tiles1, _ = _bound(cfg, 1)                           # existing path, general kernel (what the new entry launches)
        cases.append((cfg, g, tiles, D, g1))
    out = torch.full((4,), -1.0, dtype=torch.float64, device="cuda:0")
    warn = torch.full((4,), -1, dtype=torch.int32, device="cuda:0")
    torch.cuda.synchronize()

    def call(k, slot):
        cfg, g, tiles, D, _ = cases[k]
        batl.stable_dt_static(tiles, D, g.n_blocks, gamma=cfg["gamma"], cfl=cfg["cfl"], limiter_beta=cfg["limiter_beta"],
                              n_order=cfg.get("n_order", 2), flux_type=cfg.get("flux_type", 0),
                              use_divb_source=cfg["use_divb_source"], out_dt=out[slot:slot + 1],
                              out_warn=warn[slot:slot + 1])

    call(0, 0)                                                   # first call on this device: looks up the array's address
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    call(1, 1)                                                   # calls in a row on one stream, nothing in between
    call(0, 2)
    call(1, 3)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0                 # no device memory was taken by the calls
    got = out.cpu().numpy()
    assert (warn.cpu().numpy() == 0).all()

    ref = []
    for cfg, g, tiles, D, g1 in cases:
        _, _, dt = g.step(1)                                     # dt of step 0 = min dt_c of the initial state (Q-T2)
        _, _, dt1 = g1.step(1)
        assert dt > 0.0 and np.isfinite(dt)
        assert abs(dt1 - dt) <= TOL * dt
        ref.append((dt, dt1))
        g.close(); g1.close()
    assert ref[1][0] > 10.0 * ref[0][0]                          # the leftover-minimum check has teeth
    for slot, k in enumerate((0, 1, 0, 1)):
        dt, dt1 = ref[k]
        assert abs(got[slot] - dt) <= TOL * dt, (slot, got[slot], dt)
        assert got[slot] == dt1, (slot, got[slot], dt1)          # same kernel, same arithmetic: same bits
    assert got[2] == got[0] and got[3] == got[1]                 # a repeated call repeats its result


@pytest.mark.gpu
def test_static_entry_point_reports_warnings_of_the_input_state():
    import torch
    import paper_2501_06717_b200 as batl
    cfg = wl.random_uniform((2, 2, 2))
    g = batl.Grid(cfg).bind()
    U = wl.initial_conserved(cfg, g.blocks())
    U[3, 0, 4, 4, 4] = -1.0                                      # a negative density in one physical cell
    g.set_state(U)
    D = torch.tensor(np.stack([wl.cell_size(cfg, b[0]) for b in g.blocks()]), dtype=torch.float64, device="cuda:0")
    out = torch.zeros(1, dtype=torch.float64, device="cuda:0")
    warn = torch.zeros(2, dtype=torch.int32, device="cuda:0")
    kw = dict(gamma=cfg["gamma"], cfl=cfg["cfl"], limiter_beta=cfg["limiter_beta"], out_dt=out)
    batl.stable_dt_static(g.state_pointers()[0] + 16, D, g.n_blocks, out_warn=warn[0:1], **kw)
    g.set_state(wl.initial_conserved(cfg, g.blocks()))           # clean state: the bits of the last call must not stick
    batl.stable_dt_static(g.state_pointers()[0] + 16, D, g.n_blocks, out_warn=warn[1:2], **kw)
    torch.cuda.synchronize()
    w = warn.cpu().numpy()
    assert w[0] & 2 and w[1] == 0                                # BATL_WARN_NEGATIVE = 2
    g.close()
