"""Pins for the oracle's source terms, B0 evaluation points, time-step bookkeeping and body faces
(CPU only).  VERDICT round 1, "What's weak" item 1: each of these functions used to rest on
GPU-equals-oracle alone.  Every expected value below is a closed form derived by hand for a special
state (stated in the docstring of the test), a cancellation that must hold to round-off, or a
convergence order; none is produced by the oracle.

  PAPER.md L172-177 (eqs 2-4, right-hand sides)    -> test_powell_source_monopole_closed_form
  Q-S2 (B0 source), Q-B1 (B0 flux), energy part    -> test_linear_b0_uniform_plasma_closed_form,
                                                      test_dipole_uniform_b1_cancellation
  where B0 is evaluated (cell centre, face centre) -> test_linear_b0_monopole_evaluation_points,
                                                      test_dipole_static_total_field_second_order
  Q-T3 (local dt kept from stage 1), Q-T2 (lag)    -> test_local_dt_*, test_global_dt_*
  Q-F3 / Q-R3 (body faces, slopes near the body)   -> test_body_*
  Q-G5 (fixed-face tie-break)                      -> test_fixed_bc_corner_lowest_face_wins
"""
import math

import numpy as np
import pytest

import workloads as wl
from util import to_global

G = 5.0 / 3.0


def _line_grid(n_cells, lo=0.0, length=1.0, **kw):
    """n_cells x 8 x 8 cells, cubic cells, periodic: a one-dimensional problem along x."""
    d = length / n_cells
    return wl._base("line", (n_cells // 8, 1, 1), (lo, 0.0, 0.0), (lo + length, 8 * d, 8 * d), **kw)


def _set_line_state(o, cfg, prim_of_x):
    """prim_of_x(x) -> [8][n] primitive profile; constant in y and z."""
    blk = o.blocks()
    W = np.zeros((o.n_blocks, 8, 8, 8, 8))
    for b, q in enumerate(blk):
        x = wl.cell_centres(cfg, q)[0]
        W[b] = prim_of_x(x)[:, None, None, :]
    o.set_primitive(W)
    return blk


def _line(cfg, blk, o):
    Gl = to_global(cfg, blk, o.get_state())
    assert np.ptp(Gl, axis=(1, 2)).max() == 0.0           # stays one-dimensional, bit for bit
    return Gl[:, 0, 0, :]


# ------------------------------------------------------------------ Powell source, eqs (2)-(4)
def test_powell_source_monopole_closed_form(orc):
    """-B div B, -u div B, -(u.B) div B on the right of eqs (2)-(4).
    State: uniform rho, p, u = (ux, uy, 0); B = (Bx(x), 0, 0) -- a field with a real divergence.
    Piecewise-constant states, one stage, fixed dt.  By hand, per face i+1/2 (L = i, R = i+1):
      mean state has B = (Bh, 0, 0), Bh = (Bx_i + Bx_{i+1})/2  =>  c_f^2 = max(gamma p / rho, Bh^2 / rho)
      F(W) = (rho ux, rho ux^2 + p - Bx^2/2, rho ux uy, 0, 0, -Bx uy, 0, ux (e + p - Bx^2/2))
      div B1 = (Bh_i - Bh_{i-1}) / dx   (Q-S1)
    and the update is U - dt/dx (F^_i - F^_{i-1}) + dt S.  B_y must stay zero: its flux difference
    + uy dBh/dx and its source - uy dBh/dx cancel; with a wrong sign it grows by 2 dt uy div B."""
    n, rho, p, ux, uy, dt = 16, 1.3, 0.7, 0.4, -0.3, 0.003
    cfg = _line_grid(n, n_stage=1, n_order=1, dt_mode=wl.DT_FIXED, dt_fixed=dt)
    o = orc.Oracle(cfg)
    xs = (np.arange(n) + 0.5) / n
    Bx = 0.6 + 0.25 * np.sin(2 * np.pi * xs) + 0.1 * np.cos(4 * np.pi * xs + 0.3)

    def prim(x):
        W = np.zeros((8, x.size))
        W[0], W[1], W[2], W[7] = rho, ux, uy, p
        W[4] = 0.6 + 0.25 * np.sin(2 * np.pi * x) + 0.1 * np.cos(4 * np.pi * x + 0.3)
        return W
    blk = _set_line_state(o, cfg, prim)
    warn, t, _ = o.step(1)
    assert warn == 0 and t == pytest.approx(dt)
    got = _line(cfg, blk, o)

    dx = 1.0 / n
    e = p / (G - 1) + 0.5 * rho * (ux * ux + uy * uy) + 0.5 * Bx * Bx
    U = np.zeros((8, n))
    U[0], U[1], U[2], U[4], U[7] = rho, rho * ux, rho * uy, Bx, e
    F = np.zeros((8, n))
    F[0] = rho * ux
    F[1] = rho * ux * ux + p - 0.5 * Bx * Bx
    F[2] = rho * ux * uy
    F[5] = -Bx * uy
    F[7] = ux * (e + p - 0.5 * Bx * Bx)
    Bh = 0.5 * (Bx + np.roll(Bx, -1))                       # face i+1/2
    c = abs(ux) + np.sqrt(np.maximum(G * p / rho, Bh * Bh / rho))
    Fh = 0.5 * (F + np.roll(F, -1, axis=1)) - 0.5 * c * (np.roll(U, -1, axis=1) - U)
    divb = (Bh - np.roll(Bh, 1)) / dx
    S = np.zeros((8, n))
    S[1] = -Bx * divb
    S[4] = -ux * divb
    S[5] = -uy * divb
    S[7] = -(ux * Bx) * divb
    expect = U - dt / dx * (Fh - np.roll(Fh, 1, axis=1)) + dt * S
    assert np.abs(divb).max() > 0.5                         # the test has teeth
    assert np.abs(got - expect).max() <= 2e-15
    assert np.abs(got[5]).max() <= 1e-17                    # B_y: flux difference and source cancel
    assert np.abs(got[3]).max() == 0.0 and np.abs(got[6]).max() == 0.0


# ----------------------------------------------------------------------- Q-S2 with a linear B0
def test_linear_b0_uniform_plasma_closed_form(orc):
    """Q-B1 / Q-S2 signs and the energy counterpart S_e = u . S.
    State: uniform rho, u, B1, p; background field B0(x) = c + g x with a general gradient g
    (non-solenoidal, non-curl-free), for which face-centred differences are exact:
    div_h B0 = tr g, (curl_h B0)_c = eps_cde g_ed.  By hand from O-5/O-6 with uniform plasma
    (no dissipation, zero slopes, div B1 = 0):
      momentum:   -div_h[(B0.B1) I - B0 B1 - B1 B0] = +B1 tr g - (g^T - g) B1, and the source
                  -B1 tr g - (curl B0) x B1 = -B1 tr g + (g^T - g) B1 cancels it exactly  => R_mom = 0
      induction:  R_B = -g u + u tr g
      energy:     R_e = -u . (g B1)      (flux part -B1.(g u) + (u.B1) tr g, source part u . S)
    The state stays uniform, so the two-stage scheme gives B1' = B1 + dt R_B and
    e' = e - dt u . (g (B1 + dt/2 R_B)).  Run on the two-level 15-leaf grid."""
    cfg = wl.uniform_state(wl.fast_wave((2, 2, 2)), prim=(1.3, 0.2, -0.1, 0.05, 0.7, -0.4, 0.3, 0.9))
    dt = 0.05
    cfg.update(dt_mode=wl.DT_FIXED, dt_fixed=dt, use_b0=1)
    rho, u, B1, p = 1.3, np.array([0.2, -0.1, 0.05]), np.array([0.7, -0.4, 0.3]), 0.9
    g = np.array([[0.011, -0.007, 0.004], [0.009, -0.005, 0.013], [-0.006, 0.002, 0.008]])
    c = np.array([0.3, -0.2, 0.5])
    assert abs(np.trace(g)) > 1e-3 and np.abs(g - g.T).max() > 1e-3
    o = orc.Oracle(cfg)
    assert o.n_blocks == 15
    o.set_b0_linear(c, g)
    o.set_primitive(wl.initial_primitive(cfg, o.blocks()))
    U0 = o.get_state()
    warn, _, _ = o.step(1)
    assert warn == 0
    U1 = o.get_state()
    RB = -g @ u + u * np.trace(g)
    B1s = B1 + 0.5 * dt * RB
    e0 = p / (G - 1) + 0.5 * rho * (u @ u) + 0.5 * (B1 @ B1)
    scale = np.abs(c).max() + 32 * np.abs(g).sum()          # |B0| over the domain
    tol = 1e-13 * scale * dt / 2.0                          # round-off of differences of O(|B0||B1|)/D with D >= 2
    assert np.array_equal(U1[:, 0], U0[:, 0])
    for a in range(3):
        assert np.abs(U1[:, 1 + a] - rho * u[a]).max() <= tol, a
        assert np.abs(U1[:, 4 + a] - (B1[a] + dt * RB[a])).max() <= tol, a
    assert np.abs(U1[:, 7] - (e0 - dt * (u @ (g @ B1s)))).max() <= tol
    # the expected changes are far above the tolerance (each mutant moves the result by O(dt |g| |B1|))
    assert abs(dt * (u @ (g @ B1s))) > 1e4 * tol and np.abs(dt * RB).min() > 1e4 * tol


def test_dipole_uniform_b1_cancellation(orc):
    """Q-S2 with the product's dipole: uniform plasma at rest with uniform B1 != 0.  The discrete
    divergence of the B0 part of the momentum flux, (B0.B1) I - B0 B1 - B1 B0, and the source
    -B1 div_h B0 - (curl_h B0) x B1 cancel identically because both use the same face-centre B0;
    u = 0 makes every other B0 term vanish.  So in one stage rho, B1 and e stay bit-identical and the
    momentum stays zero up to the round-off of the sums that cancel.  (With B1 = 0, test T2, every
    one of these terms is multiplied by zero.)"""
    cfg = wl._base("dip", (2, 2, 2), (-8,) * 3, (8,) * 3, bc=(wl.BC_FLOAT,) * 6, use_b0=1,
                   dipole_m=(30.0, -20.0, -500.0), dt_mode=wl.DT_FIXED, dt_fixed=1e-3, n_stage=1,
                   regions=[(wl.SHAPE_SPHERE, 1, (0, 0, 0, 3.0, 0, 0))], max_level=1)
    B1 = (0.7, -0.4, 0.3)
    cfg = wl.uniform_state(cfg, prim=(1.0, 0, 0, 0) + B1 + (1.0,))
    o = orc.Oracle(cfg)
    assert o.n_blocks == 64
    blk = o.blocks()
    o.set_primitive(wl.initial_primitive(cfg, blk))
    U0 = o.get_state()
    warn, _, _ = o.step(1)
    assert warn == 0
    U1 = o.get_state()
    assert np.array_equal(U1[:, 0], U0[:, 0]) and np.array_equal(U1[:, 4:7], U0[:, 4:7])
    assert np.array_equal(U1[:, 7], U0[:, 7])
    m = np.array(cfg["dipole_m"])
    worst = 0.0
    for b, q in enumerate(blk):
        x, y, z = wl.cell_centres(cfg, q)
        D = wl.cell_size(cfg, q[0])[0]
        r = np.sqrt(x[None, None, :] ** 2 + y[None, :, None] ** 2 + z[:, None, None] ** 2)
        b0 = 2.0 * np.linalg.norm(m) / np.maximum(r - D, 0.5 * D) ** 3       # bound of |B0| around the cell
        bound = 2e-14 * b0 * np.linalg.norm(B1) / D * cfg["dt_fixed"]          # round-off of O(|B0||B1|/D) sums
        worst = max(worst, (np.abs(U1[b, 1:4]).max(axis=0) / bound).max())
    assert worst <= 1.0, worst
    # teeth: the two parts that cancel are each ~1e10 round-offs large
    assert 1e-3 * 500.0 * 0.7 / 0.5 ** 4 > 1e8 * 2e-14 * 500.0


def test_linear_b0_monopole_evaluation_points(orc):
    """Where B0 is evaluated: at the FACE centre x_lo + f D for the flux and for div_h / curl_h B0,
    at the CELL centre x_lo + (i + 1/2) D for the 8-wave term -(B1 + B0) div B1 (O-5, O-6).
    State at rest, uniform rho and p, B1 = (b(x), 0, 0) periodic, B0 = (beta + alpha x, 0, 0),
    piecewise-constant states, one stage.  By hand (momentum is zero on both sides of every face,
    so its flux carries no dissipation):
      F_rho_ux(W_j; B0f) = p - b_j^2/2 - B0f b_j
      (rho ux)' = -dt/dx (F^_{i+1/2} - F^_{i-1/2}) - dt (b_i + B0(x_i)) div B1 - dt b_i alpha
      c_{i+1/2}^2 = max(gamma p, (bh + B0f)^2) / rho,  b' and e' move by Rusanov dissipation only.
    In the continuum a field B_x(x) exerts no force along x, so (rho ux)' is pure truncation
    error: it must fall by about 4 when the cell size is halved; an evaluation point shifted by
    half a cell leaves a first-order term."""
    rho, p, alpha, beta, dt, lo = 1.1, 0.8, 0.9, 0.4, 0.002, 2.0
    resid = {}
    for n in (16, 32):
        cfg = _line_grid(n, lo=lo, n_stage=1, n_order=1, dt_mode=wl.DT_FIXED, dt_fixed=dt, use_b0=1)
        o = orc.Oracle(cfg)
        o.set_b0_linear((beta, 0, 0), [[alpha, 0, 0], [0, 0, 0], [0, 0, 0]])
        prof = lambda x: 0.5 + 0.3 * np.sin(2 * np.pi * (x - lo)) + 0.1 * np.cos(4 * np.pi * (x - lo))

        def prim(x):
            W = np.zeros((8, x.size))
            W[0], W[7], W[4] = rho, p, prof(x)
            return W
        blk = _set_line_state(o, cfg, prim)
        warn, _, _ = o.step(1)
        assert warn == 0
        got = _line(cfg, blk, o)
        dx = 1.0 / n
        i = np.arange(n)
        b = prof(lo + (i + 0.5) * dx)
        bp, bm = np.roll(b, -1), np.roll(b, 1)
        B0m, B0p, B0c = beta + alpha * (lo + i * dx), beta + alpha * (lo + (i + 1) * dx), beta + alpha * (lo + (i + 0.5) * dx)
        F = lambda bj, B0f: p - 0.5 * bj * bj - B0f * bj
        Fp = 0.5 * (F(b, B0p) + F(bp, B0p))
        Fm = 0.5 * (F(bm, B0m) + F(b, B0m))
        divb = (bp - bm) / (2 * dx)
        mom = -dt / dx * (Fp - Fm) - dt * (b + B0c) * divb - dt * b * alpha
        cp = np.sqrt(np.maximum(G * p, (0.5 * (b + bp) + B0p) ** 2) / rho)
        cm = np.sqrt(np.maximum(G * p, (0.5 * (bm + b) + B0m) ** 2) / rho)
        e = p / (G - 1) + 0.5 * b * b
        ep, em = np.roll(e, -1), np.roll(e, 1)
        assert np.abs(got[1] - mom).max() <= 1e-15
        assert np.abs(got[4] - (b + dt / (2 * dx) * (cp * (bp - b) - cm * (b - bm)))).max() <= 1e-15
        assert np.abs(got[7] - (e + dt / (2 * dx) * (cp * (ep - e) - cm * (e - em)))).max() <= 2e-15
        assert np.array_equal(got[0], np.full(n, rho)) and np.abs(got[[2, 3, 5, 6]]).max() == 0.0
        resid[n] = np.abs(got[1]).max() / dt
    assert 3.0 <= resid[16] / resid[32] <= 5.0, resid


@pytest.mark.slow
def test_dipole_static_total_field_second_order(orc):
    """Face-centre evaluation of the DIPOLE (Q-B1): choose B1 = B_u - B0(x_cell) so that the total
    field B0 + B1 is uniform at every cell centre; with uniform rho, u, p that is a steady state of
    ideal MHD, and the split scheme must keep it up to its truncation error: the one-step residual
    of every variable (L1 norm) falls by ~4 when the cell size is halved.  B0 taken half a cell away from the
    face centre leaves an O(D) residual (ratio ~2)."""
    m = np.array([3.0, -2.0, -40.0])
    Bu, u = np.array([0.3, 0.2, -0.4]), np.array([0.2, -0.1, 0.15])
    res = {}
    for nr in (2, 4):
        cfg = wl._base("dipstat", (nr,) * 3, (4.0, 3.0, 2.0), (8.0, 7.0, 6.0), bc=(wl.BC_FLOAT,) * 6, use_b0=1,
                       dipole_m=tuple(m), dt_mode=wl.DT_FIXED, dt_fixed=1e-3, n_stage=1)
        o = orc.Oracle(cfg)
        blk = o.blocks()
        W = np.zeros((o.n_blocks, 8, 8, 8, 8))
        keep = np.zeros((o.n_blocks, 8, 8, 8), dtype=bool)
        for b, q in enumerate(blk):
            x, y, z = wl.cell_centres(cfg, q)
            X = x[None, None, :] + 0 * y[None, :, None] + 0 * z[:, None, None]
            Y, Z = 0 * X + y[None, :, None], 0 * X + z[:, None, None]
            r2 = X * X + Y * Y + Z * Z
            md = m[0] * X + m[1] * Y + m[2] * Z
            for a, Xa in enumerate((X, Y, Z)):                # textbook dipole (3 (m.x) x / r^2 - m) / r^3
                W[b, 4 + a] = Bu[a] - (3.0 * md * Xa / r2 - m[a]) / r2 ** 1.5
                W[b, 1 + a] = u[a]
            W[b, 0], W[b, 7] = 1.0, 0.8
            keep[b] = (np.abs(X - 6.0) < 1.0) & (np.abs(Y - 5.0) < 1.0) & (np.abs(Z - 4.0) < 1.0)   # away from the float boundary
        o.set_primitive(W)
        U0 = o.get_state()
        warn, _, _ = o.step(1)
        assert warn == 0
        dU = (o.get_state() - U0) / cfg["dt_fixed"]
        # L1 norm: on the surfaces where a component of B1 has an extremum the limiter drops to first
        # order (O(D) error on an O(D) fraction of the cells), which the maximum norm would show
        res[nr] = np.array([np.abs(dU[:, sl][np.broadcast_to(keep[:, None], dU[:, sl].shape)]).mean()
                            for sl in (slice(1, 4), slice(4, 7), slice(7, 8))])
    ratio = res[2] / res[4]
    assert np.all(ratio >= 3.0) and np.all(ratio <= 5.5), (res, ratio)


# --------------------------------------------------------------------------- Q-T3 and Q-T2
def _euler_line(n, **kw):
    """Uniform u = (ux, 0, 0) and p, B = 0, varying rho, piecewise-constant states.  By hand
    (as in test_one_stage_first_order_density_advection_closed_form): u and p stay uniform under
    any first-order Rusanov update, so only rho moves:
      F^_{i+1/2} = ux (r_i + r_{i+1})/2 - c_{i+1/2} (r_{i+1} - r_i)/2,  c = |ux| + sqrt(gamma p / ((r_i + r_{i+1})/2))
      dt_c,i = CFL / (max(c_{i-1/2}, c_{i+1/2})/dx + 2 sqrt(gamma p / r_i)/dx)     (O-8; y and z faces see the cell itself)"""
    cfg = _line_grid(n, n_order=1, cfl=0.7, **kw)
    xs = (np.arange(n) + 0.5) / n
    rho0 = 1.0 + 0.4 * np.sin(2 * np.pi * xs) + 0.15 * np.cos(6 * np.pi * xs)
    return cfg, rho0


UX, P0 = 0.6, 0.9


def _rusanov_rho_flux(r):
    rb = 0.5 * (r + np.roll(r, -1))
    c = abs(UX) + np.sqrt(G * P0 / rb)
    return 0.5 * UX * (r + np.roll(r, -1)) - 0.5 * c * (np.roll(r, -1) - r), c


def _dt_c(r, n, cfl):
    _, c = _rusanov_rho_flux(r)
    dx = 1.0 / n
    return cfl / (np.maximum(c, np.roll(c, 1)) / dx + 2.0 * np.sqrt(G * P0 / r) / dx)


def _euler_prim(rho_of_x):
    def prim(x):
        W = np.zeros((8, x.size))
        W[0], W[1], W[7] = rho_of_x(x), UX, P0
        return W
    return prim


RHO_OF_X = lambda x: 1.0 + 0.4 * np.sin(2 * np.pi * x) + 0.15 * np.cos(6 * np.pi * x)


def test_local_dt_kept_from_stage_one_closed_form(orc):
    """Q-T3: dt_c of the cell comes from the speeds of stage 1 (the step's initial state), is
    stored, and stage 2 uses the stored value: after one two-stage step get_dt_local() is the
    closed-form dt_c of U^n (not of U*), and rho^{n+1}_i = rho_i - dt_c,i/dx (F^*_{i+1/2} - F^*_{i-1/2})
    with F^* from rho*_i = rho_i - dt_c,i/(2 dx) (F^_{i+1/2} - F^_{i-1/2})."""
    n = 16
    cfg, rho0 = _euler_line(n, dt_mode=wl.DT_LOCAL)
    o = orc.Oracle(cfg)
    blk = _set_line_state(o, cfg, _euler_prim(RHO_OF_X))
    warn, t, _ = o.step(1)
    assert warn == 0 and t == 0.0
    dtc = _dt_c(rho0, n, 0.7)
    got_dt = o.get_dt_local()
    Gdt = np.zeros((8, 8, n))
    for b, q in enumerate(blk):
        Gdt[:, :, 8 * q[1]:8 * q[1] + 8] = got_dt[b]
    assert np.ptp(Gdt, axis=(0, 1)).max() == 0.0
    assert np.abs(Gdt[0, 0] / dtc - 1.0).max() <= 4e-16
    F0, _ = _rusanov_rho_flux(rho0)
    rs = rho0 - 0.5 * dtc * n * (F0 - np.roll(F0, 1))
    assert np.abs(_dt_c(rs, n, 0.7) / dtc - 1.0).max() > 1e-3        # dt_c of U* is a different number
    Fs, _ = _rusanov_rho_flux(rs)
    expect = rho0 - dtc * n * (Fs - np.roll(Fs, 1))
    got = _line(cfg, blk, o)
    assert np.abs(got[0] - expect).max() <= 1e-15
    assert np.abs(got[1] - expect * UX).max() <= 1e-15


def test_global_dt_stage0_pass_and_lag_closed_form(orc):
    """Q-T2: dt of step 0 is the minimum of dt_c over the initial state (stage-0 pass); dt of step 1
    is the minimum of dt_c over the faces of stage 2 of step 0, whose input is
    U* = U^0 + dt_0/2 R(U^0) -- not U^0 and not U^1."""
    n = 16
    cfg, rho0 = _euler_line(n, dt_mode=wl.DT_GLOBAL)
    o = orc.Oracle(cfg)
    blk = _set_line_state(o, cfg, _euler_prim(RHO_OF_X))
    _, t0, dt0 = o.step(1)
    e0 = _dt_c(rho0, n, 0.7).min()
    assert dt0 == pytest.approx(e0, rel=4e-16) and t0 == pytest.approx(e0, rel=4e-16)
    F0, _ = _rusanov_rho_flux(rho0)
    rs = rho0 - 0.5 * e0 * n * (F0 - np.roll(F0, 1))
    Fs, _ = _rusanov_rho_flux(rs)
    r1 = rho0 - e0 * n * (Fs - np.roll(Fs, 1))
    assert np.abs(_line(cfg, blk, o)[0] - r1).max() <= 1e-15
    _, t1, dt1 = o.step(1)
    e1 = _dt_c(rs, n, 0.7).min()
    assert dt1 == pytest.approx(e1, rel=1e-14) and t1 == pytest.approx(e0 + e1, rel=1e-14)
    # the alternatives are different numbers
    assert abs(_dt_c(rho0, n, 0.7).min() / e1 - 1.0) > 1e-4 and abs(_dt_c(r1, n, 0.7).min() / e1 - 1.0) > 1e-4


# ----------------------------------------------------------------------- Q-F3 / Q-R3: the body
def _body_cfg(**kw):
    return wl._base("body", (2, 2, 2), (-4.0,) * 3, (4.0,) * 3, use_body=1, r_body=1.2, dt_mode=wl.DT_FIXED,
                    dt_fixed=0.01, n_stage=1, **kw)


def _body_global(cfg):
    x = -4.0 + (np.arange(16) + 0.5) * 0.5
    Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
    return X, Y, Z, (X * X + Y * Y + Z * Z) < cfg["r_body"] ** 2


def _run_global(orc, cfg, Wg):
    from util import from_global
    o = orc.Oracle(cfg)
    blk = o.blocks()
    o.set_primitive(from_global(cfg, blk, Wg))
    U0 = to_global(cfg, blk, o.get_state())
    warn, _, _ = o.step(1)
    assert warn == 0
    return U0, to_global(cfg, blk, o.get_state())


def _nbr(mask, axis, shift):
    return np.roll(mask, shift, axis=axis)


def test_body_face_fixed_density_closed_form(orc):
    """Q-F3: the body side of a face between a body cell and a true cell holds (rho_body, -u, B1, p)
    (p_body if given) built from the true-side face state; faces inside the body are skipped; body
    cells are never updated.  Gas at rest, uniform rho0, p0, B = 0: only the density dissipation
    -c (rho_R - rho_L)/2 with c = sqrt(gamma pbar / rhobar) of the mean state acts, so a true cell
    with m body faces gets rho' = rho0 - m dt c (rho0 - rho_body) / (2 D); the wall pressure is
    (p_body + p0)/2, so momentum moves only if p_body is given."""
    rho0, p0, rb, D = 1.0, 0.6, 3.0, 0.5
    for p_body in (-1.0, 0.25):
        cfg = _body_cfg(rho_body=rb, p_body=p_body)
        X, Y, Z, body = _body_global(cfg)
        assert 8 < body.sum() < 100
        Wg = np.zeros((8, 16, 16, 16))
        Wg[0], Wg[7] = rho0, p0
        U0, U1 = _run_global(orc, cfg, Wg)
        dt = cfg["dt_fixed"]
        pw = p0 if p_body <= 0 else p_body
        c = math.sqrt(G * (0.5 * (p0 + pw)) / (0.5 * (rho0 + rb)))
        m = sum(_nbr(body, ax, s).astype(int) for ax in (0, 1, 2) for s in (1, -1))
        expect = np.where(body, rho0, rho0 - m * dt * c * (rho0 - rb) / (2 * D))
        assert np.abs(U1[0] - expect).max() <= 1e-15
        assert (m[~body] > 0).sum() > 20
        # momentum: -dt/D (F_plus - F_minus) with wall pressure (pw + p0)/2 at body faces, p0 elsewhere
        for a, ax in ((0, 2), (1, 1), (2, 0)):                 # arrays are [z][y][x]
            plus, minus = _nbr(body, ax, -1), _nbr(body, ax, 1)   # body on the + / - side along this axis
            Fp = np.where(plus, 0.5 * (p0 + pw), p0)
            Fm = np.where(minus, 0.5 * (p0 + pw), p0)
            expect_m = np.where(body, 0.0, -dt / D * (Fp - Fm))
            assert np.abs(U1[1 + a] - expect_m).max() <= 1e-16
        # energy: e' = e - dt/D sum(F_e), F_e = -c (e_R - e_L)/2 at body faces
        eb, e0 = pw / (G - 1), p0 / (G - 1)
        expect_e = np.where(body, e0, e0 - m * dt * c * (e0 - eb) / (2 * D))
        assert np.abs(U1[7] - expect_e).max() <= 1e-15
        assert np.array_equal(U1[:, body], U0[:, body])


def test_body_face_reflects_velocity_closed_form(orc):
    """Q-F3: the body state carries -u.  Uniform flow u = (ux, 0, 0) with rho_body = rho0: the mass
    flux through a body face is exactly zero (a reflecting wall), rho ux elsewhere, so a true cell
    with the body on its -x side loses dt rho0 ux / D, on its +x side gains it.  Wall momentum
    flux: rho0 ux^2 + p -+ c rho0 ux with c = sqrt(gamma p / rho0) (the mean velocity is zero)."""
    rho0, p0, ux, D = 1.4, 0.7, 0.3, 0.5
    cfg = _body_cfg(rho_body=rho0)
    X, Y, Z, body = _body_global(cfg)
    Wg = np.zeros((8, 16, 16, 16))
    Wg[0], Wg[1], Wg[7] = rho0, ux, p0
    U0, U1 = _run_global(orc, cfg, Wg)
    dt = cfg["dt_fixed"]
    plus, minus = _nbr(body, 2, -1), _nbr(body, 2, 1)
    Fp = np.where(plus, 0.0, rho0 * ux)
    Fm = np.where(minus, 0.0, rho0 * ux)
    expect = np.where(body, rho0, rho0 - dt / D * (Fp - Fm))
    assert np.abs(U1[0] - expect).max() <= 1e-15
    assert (plus & ~body).sum() > 5 and (minus & ~body).sum() > 5
    c = math.sqrt(G * p0 / rho0)
    f0 = rho0 * ux * ux + p0
    Mp = np.where(plus, f0 + c * rho0 * ux, f0)
    Mm = np.where(minus, f0 - c * rho0 * ux, f0)
    # -u reverses the tangential velocity too: a y or z body face carries the x momentum flux
    # -+ c (rho0 (-ux) - rho0 ux)/2 = +- c rho0 ux, i.e. each such face removes dt c rho0 ux / D
    m_t = sum(_nbr(body, ax, sh).astype(int) for ax in (0, 1) for sh in (1, -1))
    expect_m = np.where(body, rho0 * ux, rho0 * ux - dt / D * (Mp - Mm) - m_t * dt / D * c * rho0 * ux)
    assert np.abs(U1[1] - expect_m).max() <= 1e-15
    assert (m_t[~body] > 0).sum() > 10
    assert np.array_equal(U1[:, body], U0[:, body])


def test_body_slopes_zero_next_to_body_cells(orc):
    """Q-R3: the limited slope of a cell is zero if c-1, c or c+1 along the sweep direction is a body
    cell.  Gas at rest with rho linear in x (second-order scheme): away from the body a linear
    profile is reconstructed exactly and nothing moves; where a slope is zeroed the face sees a jump
    of s D / 2 per zeroed side and the Rusanov dissipation -c jump / 2 moves the density.  Checked
    on every true cell whose y and z neighbours are true cells (so only x faces matter)."""
    p0, s, D, rb = 0.6, 0.05, 0.5, 2.0
    cfg = _body_cfg(rho_body=rb, n_order=2, bc=(wl.BC_FLOAT,) * 6)
    X, Y, Z, body = _body_global(cfg)
    rho = 2.0 + s * X
    Wg = np.zeros((8, 16, 16, 16))
    Wg[0], Wg[7] = rho, p0
    U0, U1 = _run_global(orc, cfg, Wg)
    dt = cfg["dt_fixed"]
    zero = body | _nbr(body, 2, 1) | _nbr(body, 2, -1)          # slope along x zeroed
    sl = np.where(zero, 0.0, s * D)
    rL, rR = rho + 0.5 * sl, rho - 0.5 * sl                     # W^L of the cell's +x face, W^R of its -x face
    # face i+1/2 between cell i (L) and i+1 (R), arrays indexed by the left cell
    L, R = rL, np.roll(rR, -1, axis=2)
    bL, bR = body, np.roll(body, -1, axis=2)
    L = np.where(bL, rb, L)
    R = np.where(bR, rb, R)
    F = -0.5 * np.sqrt(G * p0 / (0.5 * (L + R))) * (R - L)
    F = np.where(bL & bR, 0.0, F)
    expect = rho - dt / D * (F - np.roll(F, 1, axis=2))
    ok = ~body
    for ax in (0, 1):
        ok &= ~_nbr(body, ax, 1) & ~_nbr(body, ax, -1)
    ok[:, :, [0, 1, 14, 15]] = False                            # stay away from the float boundary
    assert np.abs(U1[0] - expect)[ok].max() <= 1e-15
    far = ok & ~zero & ~_nbr(zero, 2, 1) & ~_nbr(zero, 2, -1)
    assert np.array_equal(U1[0][far], U0[0][far])               # exact linear reconstruction: no flux at all
    near = ok & zero
    assert near.sum() > 10 and np.abs(U1[0] - U0[0])[near].min() > 1e-6


# ------------------------------------------------------------------------------------ Q-G5
def test_fixed_bc_corner_lowest_face_wins(orc):
    """Q-G5 (a documented reading, nothing in the paper decides it): a ghost cell outside two
    fixed faces takes the state of the face with the lower index; fixed beats float."""
    bc_prim = np.zeros((6, 8))
    for f in range(6):
        bc_prim[f] = (1.0 + f, 0, 0, 0, 0, 0, 0, 1.0)
    cfg = wl._base("corner", (1, 1, 1), (0, 0, 0), (1, 1, 1), bc=(wl.BC_FIXED, wl.BC_FLOAT, wl.BC_FIXED, wl.BC_FIXED, wl.BC_FLOAT, wl.BC_FIXED),
                   bc_prim=bc_prim)
    cfg = wl.uniform_state(cfg, prim=(9.0, 0, 0, 0, 0, 0, 0, 1.0))
    o = orc.Oracle(cfg)
    o.set_primitive(wl.initial_primitive(cfg, o.blocks()))
    S = o.get_state(with_ghost=True)[0, 0]                      # rho, [k][j][i] with 2 ghosts
    assert S[5, 5, 0] == 1.0                                    # -x face (0) alone
    assert S[5, 0, 0] == 1.0 and S[5, 11, 0] == 1.0            # -x beats -y (2) and +y (3)
    assert S[5, 0, 5] == 3.0 and S[5, 11, 5] == 4.0
    assert S[11, 11, 5] == 4.0                                  # +y (3) beats +z (5)
    assert S[11, 5, 11] == 6.0 and S[0, 5, 11] == 9.0          # fixed +z beats float +x; float/float clamps to the cell
