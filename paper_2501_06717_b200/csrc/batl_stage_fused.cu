// Fused stage kernel (steps a5-a9, and the same-level part of a1): reconstruction + Rusanov or
// HLL-type flux + 8-wave and B0 sources + update + dt minimum in one pass, and the result written
// both into the block and into the face ghosts of its same-level neighbours (row f2).  Face states
// and fluxes never leave the SM (the paper's GPU code passes them through global Flux_V[XYZ]B
// arrays, Alg. 2 L76, L82-84).  Compile-time variants cover the B0 split, local time
// stepping, first-order face states, body cells, block lists and the resolution-change operators
// (DESIGN.md section 6.1).
//
// Work decomposition (sm_100a, 148 SMs, 228 KB shared memory per SM):
//   * the unit of work is a HALF block: 8 x 8 x 4 physical cells.  The kernel is
//     persistent: two CTAs per SM, each walking the half blocks t = blockIdx.x,
//     blockIdx.x + gridDim.x, ...
//   * the tile arrives by THREE 5-D TMA tensor copies (UTMALDG) that carry all 8
//     variables each: M = 12 x 12 x 4 stored cells (x and y ghosts in line with the
//     physical cells, so x and y neighbours are plain +-1 / +-12 offsets) and the two
//     z ghost slabs of 8 x 8 x 2.  The request for the NEXT half block is issued as soon
//     as the last slope of the current one has been taken (middle of the z sweep), so its
//     HBM latency hides behind the z fluxes, the update and the stores.
//   * 256 "cell" threads own one physical cell each for all three sweeps and carry its
//     updated state U^n + f dt R in registers; 64 "helper" threads do the slopes of the
//     ghost cells next to the block faces and the fluxes of the low boundary faces.
//   * per sweep: every cell computes ONE limited slope per variable, keeps W^L of its
//     high face in registers and hands W^R of its low face to the neighbour through
//     shared memory; the flux of a face is computed once, by the thread left of it.
//   * shared-memory bandwidth is the first limit of this kernel, so the rows
//     of a half warp are chosen two apart (pitch 12 doubles: rows j and j+2 fall on
//     disjoint banks) and nothing is staged that a register can hold.
#include <cuda.h>

#include <atomic>
#include <mutex>
#include <vector>

#include "batl_device.cuh"
#include "mhd_physics.cuh"

namespace batl {
namespace {

constexpr int FT = 320;                 // threads per CTA: 256 cell threads + 64 helpers
constexpr int HK = 4;                   // physical k planes per CTA
constexpr int NPH = 256;                // physical cells of a half block
constexpr int MROW = NS;                // 12 doubles per row of M
constexpr int MPLANE = NS * NS;         // 144 per k plane
constexpr int MV = MPLANE * HK;         // 576 cells of M per variable
constexpr int ZV = NI * NI * NG;        // 128 cells of a z ghost slab per variable
constexpr int NSLOT = 320;              // face slots per sweep: 256 high faces + up to 64 low boundary faces
constexpr uint32_t TILE_BYTES = (MV + 2 * ZV) * NV * sizeof(double);   // 53,248

// per-half-block scalars kept in shared memory and read by broadcast loads where needed, so
// that no register holds them across the sweeps
enum { G_INVD = 0, G_F = 3, G_X0 = 4, G_D = 7, G_N = 12 };   // 1/D_d, f (O-7), low corner, cell size

struct FusedSmem {
  double M[NV][MV];                     // primitives after the in-place conversion
  double ZM[NV][ZV];                    // planes k0-2, k0-1 (physical i, j only)
  double ZP[NV][ZV];                    // planes k0+4, k0+5
  double wr[NV][NSLOT];                 // W^R of the face in slot s
  double fx[NV][NSLOT];                 // 2 * flux of the face in slot s
  double cx[NSLOT];                     // c_max of the face in slot s
  double xl[NSLOT];                     // normal B1 component of W^L of the face in slot s
  double b0x[3][NSLOT];                 // B0 at the centre of the face in slot s (B0 variants: computed once by the
                                        // face's owner, read by the two cells next to it for Q-S2)
  double geo[2][G_N];                   // geometry of the current and of the next half block (G_* below)
  int blk[2];                           // their block ids
  int pnb[2][8];                        // their rows of push_nbr (same-level face neighbours, -1 = none)
  uint32_t bmask[2][BODY_MASK_WORDS];   // BODY variants: bit s = stored cell s of the block is a body cell (Q-F3)
  int bflag[2];                         // ... and whether the block has any
  int fcs[2][8];                        // their rows of fc_slot (flux correction, Q-G6b; -1 = not a resolution change)
  double red[8];
  unsigned long long mbar_tile;
};

// m: the state seen as [nB][8][12][144] (a k plane of 12 x 12 stored cells is one contiguous row of
// 1,152 bytes), box {144,4,8,1}; z: seen as [nB][8][12][12][12], box {8,8,2,8,1}
struct TileMaps { CUtensorMap m, z, p; };   // p: physical cells of a half block, box {8,8,4,8,1}

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void tma_load_5d(void* dst, const CUtensorMap* map, unsigned long long* mbar,
                                            int c0, int c1, int c2, int c3, int c4) {
  asm volatile(
      "cp.async.bulk.tensor.5d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6, %7}], [%2];"
      ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(mbar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4)
      : "memory");
}

// L2 prefetch of a box (no shared memory involved): HBM -> L2 a whole iteration ahead of the load
__device__ __forceinline__ void tma_prefetch_5d(const CUtensorMap* map, int c0, int c1, int c2, int c3, int c4) {
  asm volatile("cp.async.bulk.prefetch.tensor.5d.L2.global.tile [%0, {%1, %2, %3, %4, %5}];"
               ::"l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4) : "memory");
}

__device__ __forceinline__ void tma_load_4d(void* dst, const CUtensorMap* map, unsigned long long* mbar,
                                            int c0, int c1, int c2, int c3) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
      ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(mbar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
      : "memory");
}
__device__ __forceinline__ void tma_prefetch_4d(const CUtensorMap* map, int c0, int c1, int c2, int c3) {
  asm volatile("cp.async.bulk.prefetch.tensor.4d.L2.global.tile [%0, {%1, %2, %3, %4}];"
               ::"l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
}

__device__ __forceinline__ void mbar_wait(unsigned long long* mbar, uint32_t parity) {
  uint32_t done = 0;
  while (!done) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done) : "r"(smem_u32(mbar)), "r"(parity) : "memory");
  }
}

// reciprocal and reciprocal square root: hardware seed + Newton steps, <= 2 ulp.
// The IEEE division / sqrt sequences cost about twice as many FP64 issue slots, and this
// kernel sits at the FP64-pipe / HBM ridge.
__device__ __forceinline__ double fast_rcp(double x) {
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  double e = fma(-x, y, 1.0);
  y = fma(y, e, y);
  e = fma(-x, y, 1.0);
  return fma(y, e, y);
}
__device__ __forceinline__ double fast_rsqrt(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  double g = x * y, h = 0.5 * y;          // g -> sqrt(x), h -> 1/(2 sqrt(x))
  double r = fma(-g, h, 0.5);
  g = fma(g, r, g); h = fma(h, r, h);
  r = fma(-g, h, 0.5);
  h = fma(h, r, h);
  return h + h;
}
__device__ __forceinline__ double fast_sqrt(double x) {   // x >= 0
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  double g = x * y, h = 0.5 * y;
  double r = fma(-g, h, 0.5);
  g = fma(g, r, g); h = fma(h, r, h);
  r = fma(-g, g, x);                      // residual x - g^2
  g = fma(r, h, g);
  return (x > 1e-300) ? g : 0.0;
}

// half of the MC(beta) limited slope (O-4): min(beta|dm|, beta|dp|, |dm+dp|/2)/2 with the
// sign of dm, zero at extrema.  hb = beta/2.
// plain compare-and-select minimum/maximum: fmin()/fmax() carry NaN-quieting code that costs
// several extra issue slots per call; NaNs cannot be repaired here anyway (warning flags).
__device__ __forceinline__ double dmin(double a, double b) { return a < b ? a : b; }
__device__ __forceinline__ double dmax(double a, double b) { return a > b ? a : b; }

template <bool BETA2>
__device__ __forceinline__ double half_slope(double dm, double dp, double hb) {
  // |.| only ever appears as an operand modifier, so no instruction is spent on it
  const double sel = (fabs(dm) < fabs(dp)) ? dm : dp;
  // BETA2: beta = 2 (monotonised central, the default), hb = 1: one multiplication less per slope
  const double lim = dmin(BETA2 ? fabs(sel) : hb * fabs(sel), 0.25 * (fabs(dm) + fabs(dp)));
  const int hi_dm = __double2hiint(dm);
  const bool opposite = (hi_dm ^ __double2hiint(dp)) < 0;
  // copysign(lim, dm): lim >= 0, so OR-ing the sign bit of dm is enough
  const double h = __hiloint2double(__double2hiint(lim) | (hi_dm & 0x80000000), __double2loint(lim));
  return opposite ? 0.0 : h;
}

// slopes of one cell: W^L of its high face, W^R of its low face, W0 = the cell itself.
// pm / p0 / pp point at variable 0 of the cell below, the cell and the cell above along the
// sweep direction; SM / S0 / SP are the per-variable strides of the arrays they live in.
template <int SM, int S0, int SP, bool BETA2>
__device__ __forceinline__ void cell_faces(const double* __restrict__ pm, const double* __restrict__ p0,
                                           const double* __restrict__ pp, double hb,
                                           double WL[NV], double WR[NV], double W0[NV]) {
#pragma unroll
  for (int v = 0; v < NV; ++v) {
    const double w0 = p0[v * S0];
    const double h = half_slope<BETA2>(w0 - pm[v * SM], pp[v * SP] - w0, hb);
    WL[v] = w0 + h;
    WR[v] = w0 - h;
    W0[v] = w0;
  }
}

// B0 at a point (Q-B1): analytic dipole at the origin (use_b0 = 1) or a uniform field (use_b0 = 2)
__device__ __forceinline__ void b0_point(const StageArgs& a, double x, double y, double z, double B0[3]) {
  if (a.use_b0 == 2) { B0[0] = a.m[0]; B0[1] = a.m[1]; B0[2] = a.m[2]; return; }
  const double r2 = x * x + y * y + z * z;
  const double ri = fast_rsqrt(r2), ri2 = ri * ri, ri3 = ri2 * ri;      // no division, no sqrt sequence
  const double md3 = 3.0 * (a.m[0] * x + a.m[1] * y + a.m[2] * z) * ri2;
  const bool ok = r2 > 0.0;
  B0[0] = ok ? (md3 * x - a.m[0]) * ri3 : 0.0;
  B0[1] = ok ? (md3 * y - a.m[1]) * ri3 : 0.0;
  B0[2] = ok ? (md3 * z - a.m[2]) * ri3 : 0.0;
}

// physical flux (eqs (1)-(4); with B0f = B0 at the face centre, Q-B1) plus c*U, with the sign of
// c chosen by the caller: returns G = F(W) + sgn_c * U(W); the Rusanov flux is (G_L(+c) + G_R(-c)) / 2.
// ADD: G += ... (the second state is summed straight into the first one's result: every term
// becomes an FMA into the running sum, which saves the eight final additions of a face)
template <int D, bool B0, bool ADD>
__device__ __forceinline__ void flux_plus_cu(const double W[NV], const double B0f[3], double c, double inv_gm1,
                                             double G[NV]) {
  const double rho = W[0], p = W[7];
  const double un = W[1 + D], b1n = W[4 + D];
  const double bn = B0 ? b1n + B0f[D] : b1n;
  const double b2 = W[4] * W[4] + W[5] * W[5] + W[6] * W[6];
  const double ub = W[1] * W[4] + W[2] * W[5] + W[3] * W[6];
  const double u2 = W[1] * W[1] + W[2] * W[2] + W[3] * W[3];
  const double hb2 = 0.5 * b2;
  const double e = fma(p, inv_gm1, fma(0.5 * rho, u2, hb2));   // eq. (5)
  double ptot = p + hb2;
  if (B0) ptot += B0f[0] * W[4] + B0f[1] * W[5] + B0f[2] * W[6];
  const double q = un + c;                 // F + c U = (u_n + c) U + (pressure and field terms)
  const double mq = rho * q;
  G[0] = ADD ? G[0] + mq : mq;
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    G[1 + a] = fma(mq, W[1 + a], ADD ? fma(-bn, W[4 + a], G[1 + a]) : -bn * W[4 + a]);
    G[4 + a] = fma(q, W[4 + a], ADD ? fma(-bn, W[1 + a], G[4 + a]) : -bn * W[1 + a]);
    if (B0) {
      G[1 + a] = fma(-b1n, B0f[a], G[1 + a]);
      G[4 + a] = fma(un, B0f[a], G[4 + a]);
    }
  }
  G[1 + D] += ptot;
  G[7] = fma(q, e, fma(un, ptot, ADD ? fma(-ub, bn, G[7]) : -ub * bn));
}

// flux_type 1 (Q-F4): HLL with S_L = min(0, u_n - c_f), S_R = max(0, u_n + c_f) of the mean state,
//   F = (S_R (F_L - S_L U_L) - S_L (F_R - S_R U_R)) / (S_R - S_L)
template <int D, bool B0, bool HLL>
__device__ __forceinline__ void face_flux2(const double WL[NV], const double WR[NV], const double B0f[3], double gamma,
                                           double inv_gm1, double F2[NV], double& cmax) {
  // wave speed of the arithmetic mean state (Q-F2); sums carry a factor 2
  const double srho = WL[0] + WR[0], sp = WL[7] + WR[7], sun = WL[1 + D] + WR[1 + D];
  double sbx = WL[4] + WR[4], sby = WL[5] + WR[5], sbz = WL[6] + WR[6];
  if (B0) { sbx = fma(2.0, B0f[0], sbx); sby = fma(2.0, B0f[1], sby); sbz = fma(2.0, B0f[2], sbz); }
  const double sbn = (D == 0) ? sbx : (D == 1) ? sby : sbz;
  // rho c_f^2 = (S + sqrt(S^2 - 4 gp bn^2)) / 2,  S = gamma p + B^2  (all of the mean state)
  const double gp = 0.5 * gamma * sp;
  const double bb = 0.25 * (sbx * sbx + sby * sby + sbz * sbz);
  const double bn2 = 0.25 * sbn * sbn;
  const double S = gp + bb;
  const double disc = dmax(fma(S, S, -4.0 * gp * bn2), 0.0);
  const double X = 0.5 * (S + fast_sqrt(disc));          // rho c_f^2
  const double rho = 0.5 * srho;
  const double cf = X * fast_rsqrt(X * rho);             // sqrt(X / rho)
  const double c = fabs(0.5 * sun) + cf;
  double GL[NV], GR[NV];
  cmax = c;
  if (HLL) {
    const double sl = dmin(0.0, 0.5 * sun - cf), sr = dmax(0.0, 0.5 * sun + cf);
    const double a2 = 2.0 * fast_rcp(sr - sl);           // F2 is twice the flux
    flux_plus_cu<D, B0, false>(WL, B0f, -sl, inv_gm1, GL);
    flux_plus_cu<D, B0, false>(WR, B0f, -sr, inv_gm1, GR);
    const double wl = a2 * sr, wr = -a2 * sl;
#pragma unroll
    for (int v = 0; v < NV; ++v) F2[v] = fma(wl, GL[v], wr * GR[v]);
    return;
  }
  flux_plus_cu<D, B0, false>(WL, B0f, c, inv_gm1, F2);
  flux_plus_cu<D, B0, true>(WR, B0f, -c, inv_gm1, F2);
}

// ---- thread <-> cell ---------------------------------------------------------------
// Cell thread tid owns physical cell (i, j, kk) with the j bits spread so that the two rows of
// a half warp are j and j+2: tid = i | j1 << 3 | j0 << 4 | j2 << 5 | kk << 6.
__device__ __forceinline__ int tid_of(int i, int j, int kk) {
  return i | (((j >> 1) & 1) << 3) | ((j & 1) << 4) | ((j >> 2) << 5) | (kk << 6);
}
__device__ __forceinline__ int m_off(int i, int j, int kk) { return (kk * NS + (j + NG)) * NS + (i + NG); }
__device__ __forceinline__ int z_off(int i, int j, int kz) { return (kz * NI + j) * NI + i; }

// Face slots of the exchange arrays (wr, fx, cx, xl), numbered per sweep so that the 16 lanes
// of a half warp hit 16 different bank pairs both at their own slot and at the slot of the face
// below (slot_minus).  c = position along the sweep direction, -1 = low boundary face.
//   x: 9 slots per row (boundary face first); the rows j and j+2 of a half warp are 8 rows apart
//   y: 8 slots per (j, kk) row group; groups ordered so that j and j+2 differ in parity
//   z: 64 slots per plane in thread order
__device__ __forceinline__ int slot_x(int c, int j, int kk) {
  const int r = ((j >> 1) & 1) * 8 + (j & 1) + 2 * (j >> 2) + 4 * (kk & 1) + 16 * (kk >> 1);
  return 9 * r + c + 1;
}
__device__ __forceinline__ int slot_y(int i, int c, int kk) {
  const int q = c + 1;                                   // 0..8
  return 8 * (10 * kk + 4 * (q >> 2) + ((q >> 1) & 1) + 2 * (q & 1)) + i;
}
__device__ __forceinline__ int slot_z(int i, int j, int c) { return 64 * (c + 1) + tid_of(i, j, 0); }

// Q-G6b: the thread that has computed the flux of a face on the block boundary keeps it if that boundary
// is a resolution change (fcs = the block's row of fc_slot).  (ci, cj, ck) = left cell of the face,
// low = the face is the low boundary face of the tile, kz0 = block-local k of the tile's first plane.
template <int D>
__device__ __forceinline__ void keep_boundary_flux(const StageArgs& a, const int* fcs, int ci, int cj, int ck, bool low,
                                                   const double F2[NV]) {
  const int cd = (D == 0) ? ci : (D == 1) ? cj : ck;       // -1: low block face, 7: high block face
  if (cd != -1 && cd != NI - 1) return;
  (void)low;
  const int slot = fcs[2 * D + (cd == -1 ? 0 : 1)];
  if (slot < 0) return;
  const int t_lo = (D == 0) ? cj : ci, t_hi = (D == 2) ? cj : ck;
  double* __restrict__ o = a.fc_buf + (size_t)slot * NV * NI * NI + t_hi * NI + t_lo;
#pragma unroll
  for (int v = 0; v < NV; ++v) o[v * NI * NI] = 0.5 * F2[v];   // F2 is twice the flux
}
// div0, cx0..cz0: discrete divergence and curl of B0 from its face-centre values (Q-S2), summed over the sweeps
struct SweepAcc { double divb; double speed; double div0, cx0, cy0, cz0; };

// One direction sweep of the half block (see the header comment).  hinv = 1 / (2 D_d); U is the
// running state U^n + f R of the cell (cell threads only); f = dt/2 or dt.
// The z sweep (D = 2) is the last one: once its slopes are taken the tile is dead, `tile_dead`
// runs right after the barrier (it requests the next tile), and the 8-wave source (O-6) is
// applied there, while the cell-centre u and B1 are still in registers.  div B1 needs only the
// normal field of the face states (Q-S1), which is known before any flux is.
// B0: B = B0 + B1 split (Q-B1, Q-S2); LDT: local time stepping, f differs from cell to cell
// (f_cell).  kz0 = block-local k index of plane kk = 0.
// BODY (Q-F3, Q-R3; bm = body mask of the block's 12^3 stored cells, nullptr if it has none): zero slope
// where c-1, c or c+1 is a body cell; a face with one body cell takes (rho_body, -u, B1, p) of the true
// side's face state on the body side; faces inside the body carry nothing; body cells are not updated.
template <int D, bool ACCUM, bool BETA2, bool B0, bool LDT, bool HLL, bool FC, bool BODY, class Hook>
__device__ __forceinline__ void sweep(FusedSmem& s, int tid, int i, int j, int kk, const StageArgs& a,
                                      const double* __restrict__ geo, const int* __restrict__ fcs,
                                      const uint32_t* __restrict__ bm, int kz0, double f_cell,
                                      double U[NV], SweepAcc& acc, Hook&& tile_dead) {
  auto isb = [&](int ci, int cj, int ck) -> bool {          // block-local cell, ghosts included
    const int sx = ((ck + NG) * NS + (cj + NG)) * NS + (ci + NG);
    return (bm[sx >> 5] >> (sx & 31)) & 1u;
  };
  constexpr int EX = (D == 0), EY = (D == 1), EZ = (D == 2);
  bool bL = false, bR = false, bM = false;                // body flags: left cell of the own face, right cell, cell below the left one
  const double hb = a.half_beta, gamma = a.gamma, inv_gm1 = a.inv_gm1;
  const int use_divb = a.use_divb;
  int fi = i, fj = j, fk = kk + kz0;                     // left cell of the face this thread owns
  const double* __restrict__ M = &s.M[0][0];
  const double* __restrict__ ZM = &s.ZM[0][0];
  const double* __restrict__ ZP = &s.ZP[0][0];
  double* __restrict__ wr = &s.wr[0][0];
  double* __restrict__ fx = &s.fx[0][0];
  double WL[NV], WR[NV], W0[NV];
  int my_slot = 0, slot_minus = 0;
  bool has_face = true;
  if (tid < NPH) {
    const int m0 = m_off(i, j, kk);
    if (D == 0) {
      cell_faces<MV, MV, MV, BETA2>(M + m0 - 1, M + m0, M + m0 + 1, hb, WL, WR, W0);
      my_slot = slot_x(i, j, kk);
      slot_minus = my_slot - 1;
    } else if (D == 1) {
      cell_faces<MV, MV, MV, BETA2>(M + m0 - MROW, M + m0, M + m0 + MROW, hb, WL, WR, W0);
      my_slot = slot_y(i, j, kk);
      slot_minus = slot_y(i, j - 1, kk);
    } else {
      if (kk == 0) cell_faces<ZV, MV, MV, BETA2>(ZM + z_off(i, j, 1), M + m0, M + m0 + MPLANE, hb, WL, WR, W0);
      else if (kk == HK - 1) cell_faces<MV, MV, ZV, BETA2>(M + m0 - MPLANE, M + m0, ZP + z_off(i, j, 0), hb, WL, WR, W0);
      else cell_faces<MV, MV, MV, BETA2>(M + m0 - MPLANE, M + m0, M + m0 + MPLANE, hb, WL, WR, W0);
      my_slot = slot_z(i, j, kk);
      slot_minus = my_slot - 64;
    }
    if (BODY && bm) {
      bL = isb(fi, fj, fk); bR = isb(fi + EX, fj + EY, fk + EZ); bM = isb(fi - EX, fj - EY, fk - EZ);
      if (bL | bR | bM) {
#pragma unroll
        for (int v = 0; v < NV; ++v) { WL[v] = W0[v]; WR[v] = W0[v]; }
      }
    }
#pragma unroll
    for (int v = 0; v < NV; ++v) wr[v * NSLOT + slot_minus] = WR[v];
    s.xl[my_slot] = WL[4 + D];
  } else {
    // helpers: W^L of the ghost cell below each low boundary face (and later the flux of that
    // face), W^R of the ghost cell above each high boundary face.  In x and y the two kinds
    // alternate in groups of 8 lanes, which halves the bank conflicts of the column reads.
    const int p = tid - NPH;
    double dummy[NV];
    if (D == 2) {
      const int gi = p & 7, gj = p >> 3;
      cell_faces<ZV, ZV, MV, BETA2>(ZM + z_off(gi, gj, 0), ZM + z_off(gi, gj, 1), M + m_off(gi, gj, 0), hb, WL, dummy, W0);
      my_slot = slot_z(gi, gj, -1);
      fi = gi; fj = gj; fk = kz0 - 1;
      if (BODY && bm) {
        bL = isb(gi, gj, kz0 - 1); bR = isb(gi, gj, kz0);
        if (bL | bR | isb(gi, gj, kz0 - 2)) {
#pragma unroll
          for (int v = 0; v < NV; ++v) WL[v] = W0[v];
        }
      }
      s.xl[my_slot] = WL[4 + D];
      cell_faces<MV, ZV, ZV, BETA2>(M + m_off(gi, gj, HK - 1), ZP + z_off(gi, gj, 0), ZP + z_off(gi, gj, 1), hb, dummy, WR, W0);
      if (BODY && bm) {
        if (isb(gi, gj, kz0 + HK - 1) | isb(gi, gj, kz0 + HK) | isb(gi, gj, kz0 + HK + 1)) {
#pragma unroll
          for (int v = 0; v < NV; ++v) WR[v] = W0[v];
        }
      }
      const int slot = slot_z(gi, gj, HK - 1);
#pragma unroll
      for (int v = 0; v < NV; ++v) wr[v * NSLOT + slot] = WR[v];
    } else {
      const int side = (p >> 3) & 1;
      const int a = p & 7, b = p >> 4;                       // (j, kk) for D = 0, (i, kk) for D = 1
      constexpr int st = (D == 0) ? 1 : MROW;
      const int lowc = (D == 0) ? m_off(-1, a, b) : m_off(a, -1, b);
      const int c0 = lowc + (side ? (NI + 1) * st : 0);      // ghost cell -1 or 8 along D
      cell_faces<MV, MV, MV, BETA2>(M + c0 - st, M + c0, M + c0 + st, hb, WL, WR, W0);
      my_slot = (D == 0) ? slot_x(-1, a, b) : slot_y(a, -1, b);
      fi = (D == 0) ? -1 : a; fj = (D == 0) ? a : -1; fk = b + kz0;
      has_face = side == 0;
      if (BODY && bm) {
        const int g = side ? NI : -1;                          // the ghost cell whose slope this is, along D
        const int gi = (D == 0) ? g : a, gj = (D == 0) ? a : g;
        const bool b0 = isb(gi, gj, fk);
        if (b0 | isb(gi - EX, gj - EY, fk) | isb(gi + EX, gj + EY, fk)) {
#pragma unroll
          for (int v = 0; v < NV; ++v) { WL[v] = W0[v]; WR[v] = W0[v]; }
        }
        bL = b0; bR = isb(gi + EX, gj + EY, fk);               // used by side 0 only (face -1|0)
      }
      if (side == 0) {
        s.xl[my_slot] = WL[4 + D];
      } else {
        const int slot = (D == 0) ? slot_x(NI - 1, a, b) : slot_y(a, NI - 1, b);
#pragma unroll
        for (int v = 0; v < NV; ++v) wr[v * NSLOT + slot] = WR[v];
      }
    }
  }
  if (B0 && has_face) {                                  // B0 at the centre of the own face, once per face
    double B0f[3];
    b0_point(a, fma(fi + (D == 0 ? 1.0 : 0.5), geo[G_D + 0], geo[G_X0 + 0]),
             fma(fj + (D == 1 ? 1.0 : 0.5), geo[G_D + 1], geo[G_X0 + 1]),
             fma(fk + (D == 2 ? 1.0 : 0.5), geo[G_D + 2], geo[G_X0 + 2]), B0f);
#pragma unroll
    for (int q = 0; q < 3; ++q) s.b0x[q][my_slot] = B0f[q];
  }
  __syncthreads();
  tile_dead();
  double F2[NV], c = 0.0;
  if (has_face) {
    const double wr_own_bn = WR[4 + D];
#pragma unroll
    for (int v = 0; v < NV; ++v) WR[v] = wr[v * NSLOT + my_slot];
    const bool inside = BODY && bL && bR;              // face between two body cells: no flux, no B_n, no speed
    if (BODY && (bL != bR)) {                          // Q-F3: fixed-density reflective state on the body side
      double* Wb = bL ? WL : WR;
      const double* Wt = bL ? WR : WL;
      Wb[0] = a.rho_body;
      Wb[1] = -Wt[1]; Wb[2] = -Wt[2]; Wb[3] = -Wt[3];
      Wb[4] = Wt[4]; Wb[5] = Wt[5]; Wb[6] = Wt[6];
      Wb[7] = (a.p_body > 0.0) ? a.p_body : Wt[7];
    }
    if (tid < NPH) {                                   // Q-S1: div B1 from the face-averaged normal field
      const double hinv = 0.5 * geo[D];
      const double bn_hi = inside ? 0.0 : WL[4 + D] + WR[4 + D];
      const double bn_lo = (BODY && bM) ? 2.0 * wr_own_bn : s.xl[slot_minus] + wr_own_bn;   // low face: the body side copies B1
      acc.divb = fma(bn_hi - bn_lo, hinv, acc.divb);
      if (B0 && ACCUM) {                               // Q-S2: this direction's differences of the face-centre B0
        const double dx = (s.b0x[0][my_slot] - s.b0x[0][slot_minus]) * geo[D];
        const double dy = (s.b0x[1][my_slot] - s.b0x[1][slot_minus]) * geo[D];
        const double dz = (s.b0x[2][my_slot] - s.b0x[2][slot_minus]) * geo[D];
        if (D == 0) { acc.div0 += dx; acc.cy0 -= dz; acc.cz0 += dy; }
        if (D == 1) { acc.div0 += dy; acc.cx0 += dz; acc.cz0 -= dx; }
        if (D == 2) { acc.div0 += dz; acc.cx0 -= dy; acc.cy0 += dx; }
      }
      if (D == 2 && ACCUM) {                           // O-6: sources from the cell-centre state of the stage input
        const double f = LDT ? f_cell : geo[G_F];
        double xc[3];
        if (B0) {
          xc[0] = fma(fi + 0.5, geo[G_D + 0], geo[G_X0 + 0]);
          xc[1] = fma(fj + 0.5, geo[G_D + 1], geo[G_X0 + 1]);
          xc[2] = fma(fk + 0.5, geo[G_D + 2], geo[G_X0 + 2]);
        }
        if (use_divb) {                                // 8-wave terms, RHS of eqs (2)-(4)
          const double d = -f * acc.divb;
          const double ub = W0[1] * W0[4] + W0[2] * W0[5] + W0[3] * W0[6];
          double B0c[3] = {0.0, 0.0, 0.0};
          if (B0) b0_point(a, xc[0], xc[1], xc[2], B0c);
#pragma unroll
          for (int q = 0; q < 3; ++q) {
            U[1 + q] = fma(B0 ? W0[4 + q] + B0c[q] : W0[4 + q], d, U[1 + q]);
            U[4 + q] = fma(W0[1 + q], d, U[4 + q]);
          }
          U[7] = fma(ub, d, U[7]);
        }
        if (B0) {                                      // Q-S2: -B1 div_h B0 - (curl_h B0) x B1 from face-centre B0
          const double div0 = acc.div0, cx0 = acc.cx0, cy0 = acc.cy0, cz0 = acc.cz0;
          const double sx = -W0[4] * div0 - (cy0 * W0[6] - cz0 * W0[5]);
          const double sy = -W0[5] * div0 - (cz0 * W0[4] - cx0 * W0[6]);
          const double sz = -W0[6] * div0 - (cx0 * W0[5] - cy0 * W0[4]);
          U[1] = fma(f, sx, U[1]); U[2] = fma(f, sy, U[2]); U[3] = fma(f, sz, U[3]);
          U[7] = fma(f, W0[1] * sx + W0[2] * sy + W0[3] * sz, U[7]);
        }
      }
    }
    double B0f[3] = {0.0, 0.0, 0.0};
    if (B0) {                                          // B0 at the centre of the face (published before the barrier)
#pragma unroll
      for (int q = 0; q < 3; ++q) B0f[q] = s.b0x[q][my_slot];
    }
    if (inside) {
#pragma unroll
      for (int v = 0; v < NV; ++v) F2[v] = 0.0;
    } else {
      face_flux2<D, B0, HLL>(WL, WR, B0f, gamma, inv_gm1, F2, c);
    }
    if (FC && ACCUM && a.fc_slot) keep_boundary_flux<D>(a, fcs, fi, fj, fk, tid >= NPH, F2);
    if (ACCUM) {
#pragma unroll
      for (int v = 0; v < NV; ++v) fx[v * NSLOT + my_slot] = F2[v];
    }
    s.cx[my_slot] = c;
  }
  __syncthreads();
  if (tid < NPH) {
    const double invd = geo[D];
    if (ACCUM) {
      const double fh = (LDT ? f_cell : geo[G_F]) * (0.5 * invd);
      // the flux of the own face is read back from its slot rather than kept in registers across
      // the barrier (no spills); the difference is formed first, so that equal fluxes cancel
      // exactly and a uniform state stays uniform to the last bit
#pragma unroll
      for (int v = 0; v < NV; ++v) U[v] = fma(fx[v * NSLOT + slot_minus] - fx[v * NSLOT + my_slot], fh, U[v]);
    }
    acc.speed = fma(dmax(c, s.cx[slot_minus]), invd, acc.speed);
  }
  // keep the tile loads of the next sweep below this point: hoisted above the update they
  // push the face fluxes out of the register file (plain path: 0.4905 with, 0.4923 ms/step without;
  // the B0 variants are the other way round, config 5 0.717 with, 0.709 without)
  if (!B0) asm volatile("" ::: "memory");
}

// ---- first-order face states (n_order = 1, Q-U2) ---------------------------------------
// W^L of a face is the cell below it, W^R the cell above: both are read straight from the tile,
// so there is no slope phase, no W^R exchange and only one barrier per sweep.  Same arithmetic
// as the second-order sweep with all slopes zero.
template <int SM, int SP>
__device__ __forceinline__ void faces1(const double* __restrict__ pm, const double* __restrict__ p0,
                                       const double* __restrict__ pp, int bn, double WL[NV], double WR[NV],
                                       double& bn_lo) {
#pragma unroll
  for (int v = 0; v < NV; ++v) { WL[v] = p0[v * MV]; WR[v] = pp[v * SP]; }
  bn_lo = pm[bn * SM] + WL[bn];
}

template <int D, bool ACCUM, bool B0, bool LDT, bool HLL, bool FC, bool BODY, class Hook>
__device__ __forceinline__ void sweep1(FusedSmem& s, int tid, int i, int j, int kk, const StageArgs& a,
                                       const double* __restrict__ geo, const int* __restrict__ fcs,
                                       const uint32_t* __restrict__ bm, int kz0, double f_cell,
                                       double U[NV], SweepAcc& acc, Hook&& tile_dead) {
  auto isb = [&](int ci, int cj, int ck) -> bool {          // block-local cell, ghosts included (BODY, see sweep())
    const int sx = ((ck + NG) * NS + (cj + NG)) * NS + (ci + NG);
    return (bm[sx >> 5] >> (sx & 31)) & 1u;
  };
  constexpr int EX = (D == 0), EY = (D == 1), EZ = (D == 2);
  bool bL = false, bR = false, bM = false;                // body flags: left cell of the own face, right cell, cell below the left one
  const double* __restrict__ M = &s.M[0][0];
  const double* __restrict__ ZM = &s.ZM[0][0];
  const double* __restrict__ ZP = &s.ZP[0][0];
  double* __restrict__ fx = &s.fx[0][0];
  double WL[NV], WR[NV], bn_lo = 0.0;
  int my_slot = 0, slot_minus = 0;
  int fi = i, fj = j, fk = kk + kz0;                     // left cell of the face this thread owns
  bool has_face = true;
  if (tid < NPH) {
    const double* p0 = M + m_off(i, j, kk);
    if (D == 0) {
      faces1<MV, MV>(p0 - 1, p0, p0 + 1, 4 + D, WL, WR, bn_lo);
      my_slot = slot_x(i, j, kk); slot_minus = my_slot - 1;
    } else if (D == 1) {
      faces1<MV, MV>(p0 - MROW, p0, p0 + MROW, 4 + D, WL, WR, bn_lo);
      my_slot = slot_y(i, j, kk); slot_minus = slot_y(i, j - 1, kk);
    } else {
      if (kk == 0) faces1<ZV, MV>(ZM + z_off(i, j, 1), p0, p0 + MPLANE, 4 + D, WL, WR, bn_lo);
      else if (kk == HK - 1) faces1<MV, ZV>(p0 - MPLANE, p0, ZP + z_off(i, j, 0), 4 + D, WL, WR, bn_lo);
      else faces1<MV, MV>(p0 - MPLANE, p0, p0 + MPLANE, 4 + D, WL, WR, bn_lo);
      my_slot = slot_z(i, j, kk); slot_minus = my_slot - 64;
    }
  } else {                                               // helpers: the low boundary faces
    const int p = tid - NPH;
    if (D == 2) {
      const int gi = p & 7, gj = p >> 3;
      const double* pl = ZM + z_off(gi, gj, 1);
      const double* ph = M + m_off(gi, gj, 0);
#pragma unroll
      for (int v = 0; v < NV; ++v) { WL[v] = pl[v * ZV]; WR[v] = ph[v * MV]; }
      my_slot = slot_z(gi, gj, -1);
      fi = gi; fj = gj; fk = kz0 - 1;
    } else {
      const int q = p & 31, aa = q & 7, b = q >> 3;      // (j, kk) for D = 0, (i, kk) for D = 1
      has_face = p < 32;
      constexpr int st = (D == 0) ? 1 : MROW;
      const double* pl = M + ((D == 0) ? m_off(-1, aa, b) : m_off(aa, -1, b));
#pragma unroll
      for (int v = 0; v < NV; ++v) { WL[v] = pl[v * MV]; WR[v] = pl[v * MV + st]; }
      my_slot = (D == 0) ? slot_x(-1, aa, b) : slot_y(aa, -1, b);
      fi = (D == 0) ? -1 : aa; fj = (D == 0) ? aa : -1; fk = b + kz0;
    }
  }
  double W0b[6] = {0, 0, 0, 0, 0, 0};                     // u and B1 of the cell (z sweep: Q-S2 after the barrier)
  if (B0 && D == 2 && tid < NPH) {
#pragma unroll
    for (int q = 0; q < 6; ++q) W0b[q] = WL[1 + q];
  }
  double F2[NV], c = 0.0;
  if (BODY && bm && has_face) {
    bL = isb(fi, fj, fk); bR = isb(fi + EX, fj + EY, fk + EZ);
    if (tid < NPH) bM = isb(fi - EX, fj - EY, fk - EZ);
  }
  const bool inside = BODY && bL && bR;                  // face between two body cells: no flux, no B_n, no speed
  if (has_face) {
    if (BODY && bM) bn_lo = 2.0 * WL[4 + D];             // low face: the body side copies B1 of this cell
    if (BODY && (bL != bR)) {                            // Q-F3: fixed-density reflective state on the body side
      double* Wb = bL ? WL : WR;
      const double* Wt = bL ? WR : WL;
      Wb[0] = a.rho_body;
      Wb[1] = -Wt[1]; Wb[2] = -Wt[2]; Wb[3] = -Wt[3];
      Wb[4] = Wt[4]; Wb[5] = Wt[5]; Wb[6] = Wt[6];
      Wb[7] = (a.p_body > 0.0) ? a.p_body : Wt[7];
    }
    if (tid < NPH) {                                     // Q-S1: div B1 from the face-averaged normal field
      acc.divb = fma((inside ? 0.0 : WL[4 + D] + WR[4 + D]) - bn_lo, 0.5 * geo[D], acc.divb);
      if (D == 2 && ACCUM) {                             // O-6: sources, cell-centre state = W^L
        const double f = LDT ? f_cell : geo[G_F];
        double xc[3];
        if (B0) {
          xc[0] = fma(fi + 0.5, geo[G_D + 0], geo[G_X0 + 0]);
          xc[1] = fma(fj + 0.5, geo[G_D + 1], geo[G_X0 + 1]);
          xc[2] = fma(fk + 0.5, geo[G_D + 2], geo[G_X0 + 2]);
        }
        if (a.use_divb) {
          const double d = -f * acc.divb;
          const double ub = WL[1] * WL[4] + WL[2] * WL[5] + WL[3] * WL[6];
          double B0c[3] = {0.0, 0.0, 0.0};
          if (B0) b0_point(a, xc[0], xc[1], xc[2], B0c);
#pragma unroll
          for (int q = 0; q < 3; ++q) {
            U[1 + q] = fma(B0 ? WL[4 + q] + B0c[q] : WL[4 + q], d, U[1 + q]);
            U[4 + q] = fma(WL[1 + q], d, U[4 + q]);
          }
          U[7] = fma(ub, d, U[7]);
        }
      }
    }
    double B0f[3] = {0.0, 0.0, 0.0};
    if (B0) {
      b0_point(a, fma(fi + (D == 0 ? 1.0 : 0.5), geo[G_D + 0], geo[G_X0 + 0]),
               fma(fj + (D == 1 ? 1.0 : 0.5), geo[G_D + 1], geo[G_X0 + 1]),
               fma(fk + (D == 2 ? 1.0 : 0.5), geo[G_D + 2], geo[G_X0 + 2]), B0f);
    }
    if (B0) {                                            // read by the two cells next to the face (Q-S2)
#pragma unroll
      for (int q = 0; q < 3; ++q) s.b0x[q][my_slot] = B0f[q];
    }
    if (inside) {
#pragma unroll
      for (int v = 0; v < NV; ++v) F2[v] = 0.0;
    } else {
      face_flux2<D, B0, HLL>(WL, WR, B0f, a.gamma, a.inv_gm1, F2, c);
    }
    if (FC && ACCUM && a.fc_slot) keep_boundary_flux<D>(a, fcs, fi, fj, fk, tid >= NPH, F2);
    if (ACCUM) {
#pragma unroll
      for (int v = 0; v < NV; ++v) fx[v * NSLOT + my_slot] = F2[v];
    }
    s.cx[my_slot] = c;
  }
  __syncthreads();
  tile_dead();                                           // z sweep: every read of the tile is behind us
  if (tid < NPH) {
    const double invd = geo[D];
    if (ACCUM) {
      const double fh = (LDT ? f_cell : geo[G_F]) * (0.5 * invd);
#pragma unroll
      for (int v = 0; v < NV; ++v) U[v] = fma(fx[v * NSLOT + slot_minus] - fx[v * NSLOT + my_slot], fh, U[v]);
    }
    acc.speed = fma(dmax(c, s.cx[slot_minus]), invd, acc.speed);
    if (B0 && ACCUM) {                                   // Q-S2 from the face-centre B0 the face owners published
      const double dx = (s.b0x[0][my_slot] - s.b0x[0][slot_minus]) * invd;
      const double dy = (s.b0x[1][my_slot] - s.b0x[1][slot_minus]) * invd;
      const double dz = (s.b0x[2][my_slot] - s.b0x[2][slot_minus]) * invd;
      if (D == 0) { acc.div0 += dx; acc.cy0 -= dz; acc.cz0 += dy; }
      if (D == 1) { acc.div0 += dy; acc.cx0 += dz; acc.cz0 -= dx; }
      if (D == 2) {
        acc.div0 += dz; acc.cx0 -= dy; acc.cy0 += dx;
        const double f = LDT ? f_cell : geo[G_F];
        const double div0 = acc.div0, cx0 = acc.cx0, cy0 = acc.cy0, cz0 = acc.cz0;
        // W0 = the cell itself (first order: W^L of its high face before any body-side change)
        const double sx = -W0b[3] * div0 - (cy0 * W0b[5] - cz0 * W0b[4]);
        const double sy = -W0b[4] * div0 - (cz0 * W0b[3] - cx0 * W0b[5]);
        const double sz = -W0b[5] * div0 - (cx0 * W0b[4] - cy0 * W0b[3]);
        U[1] = fma(f, sx, U[1]); U[2] = fma(f, sy, U[2]); U[3] = fma(f, sz, U[3]);
        U[7] = fma(f, W0b[0] * sx + W0b[1] * sy + W0b[2] * sz, U[7]);
      }
    }
  }
  // the next sweep overwrites fx / cx slots that slower threads may still be reading
  __syncthreads();
}

// O-3: conserved -> primitive of one stored cell, in place (rho and B1 stay as they are).
// Returns the conserved momentum and energy in mom_e (the caller may keep them as U^n).
template <int S>
__device__ __forceinline__ void to_primitive(double* __restrict__ q, double gm1, double& rho, double& p,
                                             double mom_e[4]) {
  rho = q[0];
  const double ir = fast_rcp(rho);
  const double mx = q[1 * S], my = q[2 * S], mz = q[3 * S], e = q[7 * S];
  const double ux = mx * ir, uy = my * ir, uz = mz * ir;
  const double bx = q[4 * S], by = q[5 * S], bz = q[6 * S];
  const double ke = 0.5 * rho * (ux * ux + uy * uy + uz * uz);
  const double me = 0.5 * (bx * bx + by * by + bz * bz);
  p = gm1 * (e - ke - me);
  q[1 * S] = ux; q[2 * S] = uy; q[3 * S] = uz; q[7 * S] = p;
  mom_e[0] = mx; mom_e[1] = my; mom_e[2] = mz; mom_e[3] = e;
}

// TMA requests of one half block (block b, half h): three copies, all 8 variables each
__device__ __forceinline__ void request_tile(FusedSmem& s, const TileMaps& maps, int b, int h) {
  const int k0 = NG + HK * h;
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(&s.mbar_tile)), "r"(TILE_BYTES) : "memory");
  tma_load_4d(&s.M[0][0], &maps.m, &s.mbar_tile, 0, k0, 0, b);
  tma_load_5d(&s.ZM[0][0], &maps.z, &s.mbar_tile, NG, NG, k0 - NG, 0, b);
  tma_load_5d(&s.ZP[0][0], &maps.z, &s.mbar_tile, NG, NG, k0 + HK, 0, b);
}

// The shared-memory tile is single-buffered, so its load can only be requested late in the
// previous iteration; to keep HBM latency off that path the same boxes are pulled into L2 one
// full iteration earlier.
__device__ __forceinline__ void prefetch_tile_l2(const TileMaps& maps, int b, int h) {
  const int k0 = NG + HK * h;
  tma_prefetch_4d(&maps.m, 0, k0, 0, b);
  tma_prefetch_5d(&maps.z, NG, NG, k0 - NG, 0, b);
  tma_prefetch_5d(&maps.z, NG, NG, k0 + HK, 0, b);
}

// block of work item t (half block t & 1 of the t >> 1-th block of the list; no list = all blocks)
__device__ __forceinline__ int block_of(const StageArgs& a, int t) { return a.blocks ? a.blocks[t >> 1] : t >> 1; }

// one thread publishes the scalars of a half block in slot `ph`
template <bool B0, bool BODY = false>
__device__ __forceinline__ void publish_geometry(FusedSmem& s, const StageArgs& a, int b, int ph, double f) {
  const BlockGeom& G = a.geom[b];
  if (BODY) {                              // rare (a handful of blocks around the body): one thread copies the mask
    const bool has = a.use_body && (G.flags & 1);
    s.bflag[ph] = has;
    if (has) {
      const uint32_t* __restrict__ m = a.body_mask + (size_t)G.mask_slot * BODY_MASK_WORDS;
      for (int w = 0; w < BODY_MASK_WORDS; ++w) s.bmask[ph][w] = m[w];
    }
  }
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    s.geo[ph][G_INVD + d] = G.invD[d];
    if (B0) { s.geo[ph][G_X0 + d] = G.x0[d]; s.geo[ph][G_D + d] = G.D[d]; }   // positions only matter to B0
  }
  s.geo[ph][G_F] = f;
  s.blk[ph] = b;
  if (a.push_nbr) {
#pragma unroll
    for (int q = 0; q < 6; ++q) s.pnb[ph][q] = a.push_nbr[(size_t)b * 6 + q];
  }
  if (a.fc_slot) {
#pragma unroll
    for (int q = 0; q < 6; ++q) s.fcs[ph][q] = a.fc_slot[(size_t)b * 6 + q];
  }
}

constexpr int PUBLISHER = NPH + 32;     // lane 0 of the second helper warp: helpers convert one cell, not three

// B0 / LDT: see sweep().  With LDT (Q-T3) stage 1 sums R alone (f = 1), stores dt_c of the cell
// and finishes with U^n + dt_c/2 R; stage 2 reads dt_c back and uses f = dt_c from the start.
// LIST: the blocks come from a.blocks (their ids travel through shared memory); without it
// block = t >> 1 and the plain path carries nothing it does not need.
// AMR: an operator at resolution changes is on (second-order prolongation or flux correction): the
// intermediate state stays conserved and boundary-face fluxes are kept; without it neither costs anything
template <int STAGE, bool BETA2, bool B0, bool LDT, bool LIST, bool ORDER1, bool HLL, bool AMR, bool BODY>
__global__ void __launch_bounds__(FT, 2)
stage_fused_kernel(const __grid_constant__ TileMaps maps, const __grid_constant__ CUtensorMap base_map,
                   const StageArgs a, const int n_tiles) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  FusedSmem& s = *reinterpret_cast<FusedSmem*>(smem_raw);
  const int tid = threadIdx.x;
  // Tile order: stage 2 takes the tiles in descending order.  It reads what stage 1 has just written
  // (buffer B) and writes what the next stage 1 reads (buffer A), so each of the two starts with the
  // blocks its predecessor wrote last, which are still in the 126 MB L2 (measured: 1.3 % of the step at
  // 4,096 blocks, 1.9 % at 2,048, 0.5 % at 8,192; as a run-time switch that also alternates the steps of
  // the one-stage scheme it costs half of that again: the loop bounds are compile-time constants here).
  constexpr bool REV = STAGE == 2;
  const int stride = REV ? -(int)gridDim.x : (int)gridDim.x;
  int t = REV ? n_tiles - 1 - (int)blockIdx.x : (int)blockIdx.x;
  auto in_range = [&](int x) { return REV ? x >= 0 : x < n_tiles; };
  // buffer B (the intermediate state of the two-stage scheme) holds PRIMITIVE variables: stage 1
  // converts its result once per physical cell, stage 2 finds its whole tile, ghosts included,
  // converted already (3.25 stored cells per physical cell in a half-block tile)
  // (off when a resolution-change operator needs the conserved intermediate state: AMR variants)
  constexpr bool PRIM_IN = STAGE == 2 && !AMR, PRIM_OUT = STAGE == 1 && !AMR;

  if (tid == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(&s.mbar_tile)));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  // O-7: U = U^n + f R with f = dt/2 (stage 1) or dt (stage 2) when dt is global or fixed
  double f_all = 0.0;
  if (tid == PUBLISHER) {
    f_all = (STAGE == 0) ? 0.0 : LDT ? 1.0 : (STAGE == 1 ? 0.5 : 1.0) * a.sc->dt;
    publish_geometry<B0, BODY>(s, a, in_range(t) ? (LIST ? block_of(a, t) : t >> 1) : 0, 0, f_all);
  }
  __syncthreads();
  if (tid == 0 && in_range(t)) request_tile(s, maps, LIST ? s.blk[0] : t >> 1, t & 1);

  // cell of this thread (cell threads) and its share of the ghost cells to convert: M holds
  // 576 - 256 = 320 non-physical cells per variable, one per thread; the z slabs hold 256.
  const int i = tid & 7, j = ((tid >> 3) & 1) * 2 + ((tid >> 4) & 1) + ((tid >> 5) & 1) * 4, kk = (tid >> 6) & 3;
  int g_off;
  {
    const int gk = tid / 80, r = tid - 80 * gk;         // 80 ghost cells per plane of M
    int row, col;
    if (r < 24) { row = r / MROW; col = r - MROW * row; }
    else if (r < 48) { row = (r - 24) / MROW; col = (r - 24) - MROW * row; row += NG + NI; }
    else { const int q = r - 48; row = NG + (q >> 2); col = (q & 3) < 2 ? (q & 3) : NI + (q & 3); }
    g_off = (gk * NS + row) * NS + col;
  }
  const double INF = __longlong_as_double(0x7FF0000000000000ll);
  double dt_min = INF;
  uint32_t phase = 0;

  for (; in_range(t); t += stride, phase ^= 1) {
    const int b = LIST ? s.blk[phase] : t >> 1;
    const int kz0 = HK * (t & 1);                        // block-local k of plane kk = 0
    const int t_next = t + stride;
    const uint32_t* bm = (BODY && s.bflag[phase]) ? s.bmask[phase] : nullptr;
    bool own_body = false;
    if (BODY && bm && tid < NPH) {
      const int sx = ((kz0 + kk + NG) * NS + (j + NG)) * NS + (i + NG);
      own_body = (bm[sx >> 5] >> (sx & 31)) & 1u;
    }
    const size_t g0 = (size_t)b * BLOCK_DOUBLES + ((size_t)(NG + kz0 + kk) * NS + (j + NG)) * NS + (i + NG);
    const size_t cell = (size_t)b * NPHYS + (size_t)((kz0 + kk) * NI + j) * NI + i;   // dt_local index
    double U[NV], f_cell = 1.0;
    if (tid < NPH) {
      if (STAGE == 2) {                                  // U^n of the cell; lands while the tile is awaited
#pragma unroll
        for (int v = 0; v < NV; ++v) U[v] = a.base[g0 + (size_t)v * NCELL];
        if (LDT) f_cell = a.dt_local[cell];
      } else if (LDT) {
#pragma unroll
        for (int v = 0; v < NV; ++v) U[v] = 0.0;
      }
    }
    int b_next = 0;
    if (tid == PUBLISHER && in_range(t_next)) {                 // next half block, one iteration ahead
      b_next = LIST ? block_of(a, t_next) : t_next >> 1;
      // measured: worth 7 % for the short first-order iteration, nothing for the second-order one
      if (ORDER1) prefetch_tile_l2(maps, b_next, t_next & 1);
      // stage 2 reads U^n of the physical cells with plain loads at the top of the next iteration
      if (STAGE == 2) tma_prefetch_5d(&base_map, NG, NG, NG + HK * (t_next & 1), 0, b_next);
    }
    mbar_wait(&s.mbar_tile, phase);

    if (!PRIM_IN) {
      // ---- O-3: conserved -> primitive, in place
      double rho, p, me[4];
      to_primitive<MV>(&s.M[0][0] + g_off, a.gm1, rho, p, me);
      if (tid < NPH) {
        to_primitive<ZV>((tid < ZV ? &s.ZM[0][0] : &s.ZP[0][0]) + (tid & (ZV - 1)), a.gm1, rho, p, me);
        double* q = &s.M[0][0] + m_off(i, j, kk);
        to_primitive<MV>(q, a.gm1, rho, p, me);
        if ((STAGE == 1 || STAGE == 3) && !LDT) {        // stages 1 and 3: U^n is the stage input itself
          U[0] = rho; U[1] = me[0]; U[2] = me[1]; U[3] = me[2];
          U[4] = q[4 * MV]; U[5] = q[5 * MV]; U[6] = q[6 * MV]; U[7] = me[3];
        }
        int warn = 0;
        if (!isfinite(rho) || !isfinite(p)) warn |= BATL_WARN_NONFINITE;
        if (rho <= 0.0 || p <= 0.0) warn |= BATL_WARN_NEGATIVE;
        if (warn && !own_body) atomicOr(&a.sc->warn, warn);
      }
      __syncthreads();
      // scalars of the next half block go into the other slot only now: the slowest cell threads of
      // the previous iteration read geo[phase ^ 1] (1/D_z, f) after its last barrier, and every
      // thread has left that iteration once it has passed the barrier above
      if (tid == PUBLISHER && in_range(t_next)) publish_geometry<B0, BODY>(s, a, b_next, phase ^ 1, f_all);
    } else if (tid < NPH) {
      // stage 2: the tile holds the primitives stage 1 wrote (buffer B): no
      // conversion pass and no barrier; the warning bits come from the cell's own rho and p
      const double rho = s.M[0][m_off(i, j, kk)], p = s.M[7][m_off(i, j, kk)];
      int warn = 0;
      if (!isfinite(rho) || !isfinite(p)) warn |= BATL_WARN_NONFINITE;
      if (rho <= 0.0 || p <= 0.0) warn |= BATL_WARN_NEGATIVE;
      if (warn && !own_body) atomicOr(&a.sc->warn, warn);
    }

    const double* geo = s.geo[phase];
    SweepAcc acc;
    acc.divb = 0.0; acc.speed = 0.0;
    acc.div0 = acc.cx0 = acc.cy0 = acc.cz0 = 0.0;
    auto nothing = [] {};
    // without the conversion barrier the first barrier of the x sweep is the point at which every
    // thread has left the previous iteration
    auto publish_next = [&] {
      if (PRIM_IN && tid == PUBLISHER && in_range(t_next)) publish_geometry<B0, BODY>(s, a, b_next, phase ^ 1, f_all);
    };
    constexpr bool ACC = STAGE != 0;
    auto next_tile = [&] {
      if (tid == 0 && in_range(t_next)) {                // the tile is dead: fetch the next one
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        request_tile(s, maps, LIST ? s.blk[phase ^ 1] : t_next >> 1, t_next & 1);
      }
    };
    if (ORDER1) {
      sweep1<0, ACC, B0, LDT, HLL, AMR, BODY>(s, tid, i, j, kk, a, geo, s.fcs[phase], bm, kz0, f_cell, U, acc, publish_next);
      sweep1<1, ACC, B0, LDT, HLL, AMR, BODY>(s, tid, i, j, kk, a, geo, s.fcs[phase], bm, kz0, f_cell, U, acc, nothing);
      sweep1<2, ACC, B0, LDT, HLL, AMR, BODY>(s, tid, i, j, kk, a, geo, s.fcs[phase], bm, kz0, f_cell, U, acc, next_tile);
    } else {
      sweep<0, ACC, BETA2, B0, LDT, HLL, AMR, BODY>(s, tid, i, j, kk, a, geo, s.fcs[phase], bm, kz0, f_cell, U, acc, publish_next);
      sweep<1, ACC, BETA2, B0, LDT, HLL, AMR, BODY>(s, tid, i, j, kk, a, geo, s.fcs[phase], bm, kz0, f_cell, U, acc, nothing);
      sweep<2, ACC, BETA2, B0, LDT, HLL, AMR, BODY>(s, tid, i, j, kk, a, geo, s.fcs[phase], bm, kz0, f_cell, U, acc, next_tile);
    }

    if (tid < NPH) {
      const double dt_c = a.cfl * fast_rcp(acc.speed);   // O-8
      if (STAGE != 1 && !own_body) dt_min = dmin(dt_min, dt_c);
      if ((STAGE == 1 || STAGE == 3) && LDT && !own_body) {   // Q-T3: U* = U^n + dt_c/2 R, dt_c kept for stage 2
        a.dt_local[cell] = dt_c;
        const double h = (STAGE == 1 ? 0.5 : 1.0) * dt_c;
#pragma unroll
        for (int v = 0; v < NV; ++v) U[v] = fma(h, U[v], a.base[g0 + (size_t)v * NCELL]);
      }
      if (BODY && own_body && STAGE != 0) {                 // Q-F3: body cells are never updated
#pragma unroll
        for (int v = 0; v < NV; ++v) U[v] = a.base[g0 + (size_t)v * NCELL];
      }
      if (PRIM_OUT) {                                    // same arithmetic as to_primitive()
        const double ir = fast_rcp(U[0]);
        const double ux = U[1] * ir, uy = U[2] * ir, uz = U[3] * ir;
        const double ke = 0.5 * U[0] * (ux * ux + uy * uy + uz * uz);
        const double me = 0.5 * (U[4] * U[4] + U[5] * U[5] + U[6] * U[6]);
        U[7] = a.gm1 * (U[7] - ke - me);
        U[1] = ux; U[2] = uy; U[3] = uz;
      }
      if (STAGE != 0) {
        double* __restrict__ o = a.out + g0;
        int pn[3] = {-1, -1, -1};
        if (a.push_nbr) push_targets(s.pnb[phase], i, j, kz0 + kk, pn);
#pragma unroll
        for (int v = 0; v < NV; ++v) o[(size_t)v * NCELL] = U[v];            // O-7
        // the cell is a face ghost of up to three same-level neighbours: written here, no fill pass
        if (a.push_nbr) push_cell_t<AMR>(a, o, pn, b, i, j, kz0 + kk, U);   // AMR: prolonged pushes into finer neighbours too
      }
    }
    // no barrier here: the next iteration writes wr / xl only after its conversion barrier,
    // and every read of fx / cx above precedes that barrier in program order
  }

  // ---- a9: minimum of dt_c over everything this CTA has seen, one atomic
  if (STAGE != 1 && a.dt_mode == BATL_DT_GLOBAL) {
    if (tid >= NPH) dt_min = INF;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) dt_min = fmin(dt_min, __shfl_xor_sync(0xffffffffu, dt_min, o));
    if ((tid & 31) == 0 && tid < NPH) s.red[tid >> 5] = dt_min;
    __syncthreads();
    if (tid < 32) {
      double v = (tid < 8) ? s.red[tid] : INF;
#pragma unroll
      for (int o = 4; o > 0; o >>= 1) v = fmin(v, __shfl_xor_sync(0xffffffffu, v, o));
      if (tid == 0) atomic_min_positive(&a.sc->dt_next_bits, v);
    }
  }
}

// ---- host side: tensor maps ----------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn() {
  static EncodeTiledFn fn = nullptr;
  static std::once_flag once;
  std::call_once(once, [] {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<EncodeTiledFn>(p);
  });
  return fn;
}

// state buffer seen as a 5-D tensor [block][var][k][j][i]; one box carries all 8 variables
bool make_map(CUtensorMap* m, const double* base, int n_blocks, int bi, int bj, int bk) {
  EncodeTiledFn enc = encode_fn();
  if (!enc) return false;
  const cuuint64_t dims[5] = {NS, NS, NS, NV, (cuuint64_t)n_blocks};
  const cuuint64_t strides[4] = {NS * sizeof(double), NS * NS * sizeof(double), NCELL * sizeof(double), BLOCK_BYTES};
  const cuuint32_t box[5] = {(cuuint32_t)bi, (cuuint32_t)bj, (cuuint32_t)bk, NV, 1};
  const cuuint32_t estr[5] = {1, 1, 1, 1, 1};
  return enc(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 5, const_cast<double*>(base), dims, strides, box, estr,
             CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// whole k planes: [block][var][k][144], box = 4 planes x 8 variables
bool make_plane_map(CUtensorMap* m, const double* base, int n_blocks) {
  EncodeTiledFn enc = encode_fn();
  if (!enc) return false;
  const cuuint64_t dims[4] = {NS * NS, NS, NV, (cuuint64_t)n_blocks};
  const cuuint64_t strides[3] = {NS * NS * sizeof(double), NCELL * sizeof(double), BLOCK_BYTES};
  const cuuint32_t box[4] = {NS * NS, HK, NV, 1};
  const cuuint32_t estr[4] = {1, 1, 1, 1};
  return enc(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, const_cast<double*>(base), dims, strides, box, estr,
             CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

struct MapCacheEntry { const double* base; int n_blocks; TileMaps maps; };
std::mutex g_cache_mutex;
std::vector<MapCacheEntry> g_cache;

bool get_maps(const double* base, int n_blocks, TileMaps* out) {
  std::lock_guard<std::mutex> lock(g_cache_mutex);
  for (const auto& e : g_cache)
    if (e.base == base && e.n_blocks == n_blocks) { *out = e.maps; return true; }
  MapCacheEntry e;
  e.base = base; e.n_blocks = n_blocks;
  if (!make_plane_map(&e.maps.m, base, n_blocks)) return false;
  if (!make_map(&e.maps.z, base, n_blocks, NI, NI, NG)) return false;
  if (!make_map(&e.maps.p, base, n_blocks, NI, NI, HK)) return false;
  if (g_cache.size() >= 64) g_cache.erase(g_cache.begin());
  g_cache.push_back(e);
  *out = e.maps;
  return true;
}

}  // namespace

// Everything but blocks that hold body cells (Q-F3, Q-R3): those go to the general kernel, which
// the caller launches on its own block list.
// The HLL-type flux (Q-F4) has fused kernels for the plain path and for the full magnetosphere
// physics, second order; other combinations with it run the general kernel.
bool stage_fused_supports(const StageArgs& a) {
  if (a.flux_type == 0) return true;
  const bool b0 = a.use_b0 != 0, ldt = a.dt_mode == BATL_DT_LOCAL;
  return a.n_order != 1 && b0 == ldt;
}

namespace {
template <int STAGE, bool BETA2, bool B0, bool LDT, bool LIST, bool ORDER1, bool HLL, bool AMR, bool BODY>
cudaError_t launch_variant(int grid, const TileMaps& maps, const CUtensorMap& base_map, const StageArgs& a, int n_tiles,
                           cudaStream_t st) {
  // the attribute is per device and per instantiation: one bit per device, set once it has been
  // applied (grids of several host threads / devices may launch concurrently)
  static std::atomic<unsigned long long> ready{0};
  int dev = 0;
  cudaGetDevice(&dev);
  if (!((ready.load(std::memory_order_acquire) >> (dev & 63)) & 1ull)) {
    const cudaError_t e = cudaFuncSetAttribute(stage_fused_kernel<STAGE, BETA2, B0, LDT, LIST, ORDER1, HLL, AMR, BODY>,
                                               cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(FusedSmem));
    if (e != cudaSuccess) return e;
    ready.fetch_or(1ull << (dev & 63), std::memory_order_release);
  }
  stage_fused_kernel<STAGE, BETA2, B0, LDT, LIST, ORDER1, HLL, AMR, BODY><<<grid, FT, sizeof(FusedSmem), st>>>(maps, base_map, a, n_tiles);
  return cudaGetLastError();
}

template <bool BETA2, bool B0, bool LDT, bool LIST, bool ORDER1 = false, bool HLL = false, bool BODY = false>
cudaError_t launch_stage_of(int stage, int grid, const TileMaps& maps, const StageArgs& a, int n_tiles, cudaStream_t st) {
  TileMaps bm;
  if (!get_maps(a.base, a.n_blocks, &bm)) return cudaErrorNotSupported;
  const CUtensorMap& base_map = bm.p;
  if (stage == 0) return launch_variant<0, BETA2, B0, LDT, LIST, ORDER1, HLL, false, BODY>(grid, maps, base_map, a, n_tiles, st);
  if ((a.b_prim == 0 && stage != 3) || a.fc_slot || a.push_fine) {   // multi-level grid or resolution-change operators
    if (stage == 1) return launch_variant<1, BETA2, B0, LDT, LIST, ORDER1, HLL, true, BODY>(grid, maps, base_map, a, n_tiles, st);
    if (stage == 2) return launch_variant<2, BETA2, B0, LDT, LIST, ORDER1, HLL, true, BODY>(grid, maps, base_map, a, n_tiles, st);
    return launch_variant<3, BETA2, B0, LDT, LIST, ORDER1, HLL, true, BODY>(grid, maps, base_map, a, n_tiles, st);
  }
  if (stage == 1) return launch_variant<1, BETA2, B0, LDT, LIST, ORDER1, HLL, false, BODY>(grid, maps, base_map, a, n_tiles, st);
  if (stage == 2) return launch_variant<2, BETA2, B0, LDT, LIST, ORDER1, HLL, false, BODY>(grid, maps, base_map, a, n_tiles, st);
  return launch_variant<3, BETA2, B0, LDT, LIST, ORDER1, HLL, false, BODY>(grid, maps, base_map, a, n_tiles, st);
}
}  // namespace

// a.blocks / a.n_list: the blocks to process (nullptr = all a.n_blocks of them)
// Blocks with body cells (Q-F3, Q-R3) inside the fused kernel: built for the magnetosphere physics (B0 split,
// local time stepping, second order); other combinations leave them to the general kernel.
bool stage_fused_handles_body(const StageArgs& a) {
  return a.use_body && a.use_b0 != 0 && a.dt_mode == BATL_DT_LOCAL && !(a.n_order == 1 && a.flux_type == 1);
}

cudaError_t launch_stage_fused(int stage, const StageArgs& a, cudaStream_t st) {
  const int n_list = a.blocks ? a.n_list : a.n_blocks;
  if (n_list == 0) return cudaSuccess;
  TileMaps maps;
  if (!get_maps(a.in, a.n_blocks, &maps)) return cudaErrorNotSupported;
  const int n_sm = a.n_sm;                                   // of the device the grid is bound on (batl_bind)
  if (n_sm <= 0) return cudaErrorInvalidDevice;
  const int n_tiles = 2 * n_list;                          // half blocks
  const int grid = n_tiles < 2 * n_sm ? n_tiles : 2 * n_sm; // persistent: two CTAs per SM
  const bool b0 = a.use_b0 != 0, ldt = a.dt_mode == BATL_DT_LOCAL;
  if (a.fused_body) {                                      // every block, body cells included (config 5's physics)
    if (!stage_fused_handles_body(a) || a.blocks) return cudaErrorNotSupported;
    if (a.flux_type == 1) return launch_stage_of<false, true, true, false, false, true, true>(stage, grid, maps, a, n_tiles, st);
    if (a.n_order == 1) return launch_stage_of<false, true, true, false, true, false, true>(stage, grid, maps, a, n_tiles, st);
    return launch_stage_of<false, true, true, false, false, false, true>(stage, grid, maps, a, n_tiles, st);
  }
  if (a.flux_type == 1) {
    if (b0 && ldt) return launch_stage_of<false, true, true, true, false, true>(stage, grid, maps, a, n_tiles, st);
    return launch_stage_of<false, false, false, true, false, true>(stage, grid, maps, a, n_tiles, st);
  }
  // first-order face states have kernels of their own for the plain path and for the full
  // magnetosphere physics; other combinations run the second-order kernels with beta = 0
  if (a.n_order == 1 && b0 && ldt) return launch_stage_of<false, true, true, true, true>(stage, grid, maps, a, n_tiles, st);
  if (a.n_order == 1 && !b0 && !ldt && !a.blocks) return launch_stage_of<false, false, false, false, true>(stage, grid, maps, a, n_tiles, st);
  if (b0 && ldt) return launch_stage_of<false, true, true, true>(stage, grid, maps, a, n_tiles, st);
  if (b0) return launch_stage_of<false, true, false, true>(stage, grid, maps, a, n_tiles, st);
  if (ldt) return launch_stage_of<false, false, true, true>(stage, grid, maps, a, n_tiles, st);
  if (a.blocks) return launch_stage_of<false, false, false, true>(stage, grid, maps, a, n_tiles, st);
  // plain path; compile-time special case of the default limiter (beta = 2)
  if (a.beta == 2.0) return launch_stage_of<true, false, false, false>(stage, grid, maps, a, n_tiles, st);
  return launch_stage_of<false, false, false, false>(stage, grid, maps, a, n_tiles, st);
}

}  // namespace batl
