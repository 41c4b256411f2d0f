// Fused stage kernel (steps a5-a9) for blocks without B0 split and without body cells:
// reconstruction + Rusanov flux + 8-wave source + update + dt minimum in one pass,
// face states and fluxes never leave the SM (the paper's GPU code passes them through
// global Flux_V[XYZ]B arrays, Alg. 2 L76, L82-84).
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

struct FusedSmem {
  double M[NV][MV];                     // primitives after the in-place conversion
  double ZM[NV][ZV];                    // planes k0-2, k0-1 (physical i, j only)
  double ZP[NV][ZV];                    // planes k0+4, k0+5
  double wr[NV][NSLOT];                 // W^R of the face in slot s
  double fx[NV][NSLOT];                 // 2 * flux of the face in slot s
  double cx[NSLOT];                     // c_max of the face in slot s
  double xl[NSLOT];                     // normal B1 component of W^L of the face in slot s
  double invd[2][4];                    // 1 / D_d of the current and of the next half block
  double red[8];
  unsigned long long mbar_tile;
};

struct TileMaps { CUtensorMap m, z; };  // boxes {12,12,4,8,1} and {8,8,2,8,1} of [nB][8][12][12][12]

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void tma_load_5d(void* dst, const CUtensorMap* map, unsigned long long* mbar,
                                            int c0, int c1, int c2, int c3, int c4) {
  asm volatile(
      "cp.async.bulk.tensor.5d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6, %7}], [%2];"
      ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(mbar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4)
      : "memory");
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

// physical flux (eqs (1)-(4), B0 = 0) plus c*U, with the sign of c chosen by the caller:
// returns G = F(W) + sgn_c * U(W); the Rusanov flux is (G_L(+c) + G_R(-c)) / 2.
template <int D>
__device__ __forceinline__ void flux_plus_cu(const double W[NV], double c, double inv_gm1, double G[NV]) {
  const double rho = W[0], p = W[7];
  const double un = W[1 + D], bn = W[4 + D];
  const double b2 = W[4] * W[4] + W[5] * W[5] + W[6] * W[6];
  const double ub = W[1] * W[4] + W[2] * W[5] + W[3] * W[6];
  const double u2 = W[1] * W[1] + W[2] * W[2] + W[3] * W[3];
  const double hb2 = 0.5 * b2;
  const double e = fma(p, inv_gm1, fma(0.5 * rho, u2, hb2));   // eq. (5)
  const double ptot = p + hb2;
  const double q = un + c;                 // F + c U = (u_n + c) U + (pressure and field terms)
  const double mq = rho * q;
  G[0] = mq;
#pragma unroll
  for (int a = 0; a < 3; ++a) G[1 + a] = fma(mq, W[1 + a], -bn * W[4 + a]);
  G[1 + D] += ptot;
#pragma unroll
  for (int a = 0; a < 3; ++a) G[4 + a] = fma(q, W[4 + a], -bn * W[1 + a]);
  G[7] = fma(q, e, fma(un, ptot, -ub * bn));
}

// twice the Rusanov flux of one face (O-5), B_n sum and c_max
template <int D>
__device__ __forceinline__ void face_flux2(const double WL[NV], const double WR[NV], double gamma, double inv_gm1,
                                           double F2[NV], double& Bn2, double& cmax) {
  // wave speed of the arithmetic mean state (Q-F2); sums carry a factor 2
  const double srho = WL[0] + WR[0], sp = WL[7] + WR[7], sun = WL[1 + D] + WR[1 + D];
  const double sbx = WL[4] + WR[4], sby = WL[5] + WR[5], sbz = WL[6] + WR[6];
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
  flux_plus_cu<D>(WL, c, inv_gm1, GL);
  flux_plus_cu<D>(WR, -c, inv_gm1, GR);
#pragma unroll
  for (int v = 0; v < NV; ++v) F2[v] = GL[v] + GR[v];
  Bn2 = sbn;
  cmax = c;
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

struct SweepAcc { double divb; double speed; };

// One direction sweep of the half block (see the header comment).  hinv = 1 / (2 D_d); U is the
// running state U^n + f R of the cell (cell threads only); f = dt/2 or dt.
// The z sweep (D = 2) is the last one: once its slopes are taken the tile is dead, `tile_dead`
// runs right after the barrier (it requests the next tile), and the 8-wave source (O-6) is
// applied there, while the cell-centre u and B1 are still in registers.  div B1 needs only the
// normal field of the face states (Q-S1), which is known before any flux is.
template <int D, bool ACCUM, bool BETA2, class Hook>
__device__ __forceinline__ void sweep(FusedSmem& s, int tid, int i, int j, int kk, double hb, double gamma,
                                      double inv_gm1, const double* __restrict__ geo, int use_divb,
                                      double U[NV], SweepAcc& acc, Hook&& tile_dead) {
  // geo = {1/D_x, 1/D_y, 1/D_z, f}: read from shared memory where needed (broadcast loads),
  // so that no register holds them across the sweeps
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
      s.xl[my_slot] = WL[4 + D];
      cell_faces<MV, ZV, ZV, BETA2>(M + m_off(gi, gj, HK - 1), ZP + z_off(gi, gj, 0), ZP + z_off(gi, gj, 1), hb, dummy, WR, W0);
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
      has_face = side == 0;
      if (side == 0) {
        s.xl[my_slot] = WL[4 + D];
      } else {
        const int slot = (D == 0) ? slot_x(NI - 1, a, b) : slot_y(a, NI - 1, b);
#pragma unroll
        for (int v = 0; v < NV; ++v) wr[v * NSLOT + slot] = WR[v];
      }
    }
  }
  __syncthreads();
  tile_dead();
  double F2[NV], c = 0.0;
  if (has_face) {
    const double wr_own_bn = WR[4 + D];
#pragma unroll
    for (int v = 0; v < NV; ++v) WR[v] = wr[v * NSLOT + my_slot];
    if (tid < NPH) {                                   // Q-S1: div B1 from the face-averaged normal field
      const double hinv = 0.5 * geo[D];
      acc.divb = fma((WL[4 + D] + WR[4 + D]) - (s.xl[slot_minus] + wr_own_bn), hinv, acc.divb);
      if (D == 2 && ACCUM && use_divb) {               // O-6: 8-wave source, cell-centre state of the stage input
        const double d = -geo[3] * acc.divb;
        const double ub = W0[1] * W0[4] + W0[2] * W0[5] + W0[3] * W0[6];
#pragma unroll
        for (int q = 0; q < 3; ++q) {
          U[1 + q] = fma(W0[4 + q], d, U[1 + q]);
          U[4 + q] = fma(W0[1 + q], d, U[4 + q]);
        }
        U[7] = fma(ub, d, U[7]);
      }
    }
    double Bn2;
    face_flux2<D>(WL, WR, gamma, inv_gm1, F2, Bn2, c);
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
      const double fh = geo[3] * (0.5 * invd);
#pragma unroll
      for (int v = 0; v < NV; ++v) U[v] = fma(fx[v * NSLOT + slot_minus] - F2[v], fh, U[v]);
    }
    acc.speed = fma(dmax(c, s.cx[slot_minus]), invd, acc.speed);
  }
  // keep the tile loads of the next sweep below this point: hoisted above the update they
  // push the face fluxes out of the register file
  asm volatile("" ::: "memory");
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

// TMA requests of one half block: three copies, all 8 variables each (one thread issues them)
__device__ __forceinline__ void request_tile(FusedSmem& s, const TileMaps& maps, int t) {
  const int b = t >> 1, k0 = NG + HK * (t & 1);
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(&s.mbar_tile)), "r"(TILE_BYTES) : "memory");
  tma_load_5d(&s.M[0][0], &maps.m, &s.mbar_tile, 0, 0, k0, 0, b);
  tma_load_5d(&s.ZM[0][0], &maps.z, &s.mbar_tile, NG, NG, k0 - NG, 0, b);
  tma_load_5d(&s.ZP[0][0], &maps.z, &s.mbar_tile, NG, NG, k0 + HK, 0, b);
}

template <int STAGE, bool BETA2>
__global__ void __launch_bounds__(FT, 2)
stage_fused_kernel(const __grid_constant__ TileMaps maps, const StageArgs a, const int n_tiles) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  FusedSmem& s = *reinterpret_cast<FusedSmem*>(smem_raw);
  const int tid = threadIdx.x;
  const int stride = gridDim.x;
  int t = blockIdx.x;

  if (tid == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(&s.mbar_tile)));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (tid == 32) {                                      // 1 / D_d of the first half block
    const BlockGeom& G = a.geom[t < n_tiles ? t >> 1 : 0];
    s.invd[0][0] = G.invD[0]; s.invd[0][1] = G.invD[1]; s.invd[0][2] = G.invD[2];
    // O-7: U = U^n + f R with f = dt/2 (stage 1) or dt (stage 2); dt is global or fixed here
    s.invd[0][3] = s.invd[1][3] = (STAGE == 0) ? 0.0 : (STAGE == 1 ? 0.5 : 1.0) * a.sc->dt;
  }
  __syncthreads();
  if (tid == 0 && t < n_tiles) request_tile(s, maps, t);

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

  for (; t < n_tiles; t += stride, phase ^= 1) {
    const int b = t >> 1;
    const int k0 = NG + HK * (t & 1);                    // first physical storage plane of this half
    const int t_next = t + stride;
    const size_t g0 = (size_t)b * BLOCK_DOUBLES + ((size_t)(k0 + kk) * NS + (j + NG)) * NS + (i + NG);
    double U[NV];
    if (STAGE == 2 && tid < NPH) {                       // U^n of the cell; lands while the tile is awaited
#pragma unroll
      for (int v = 0; v < NV; ++v) U[v] = a.base[g0 + (size_t)v * NCELL];
    }
    if (tid == 32 && t_next < n_tiles) {                 // geometry of the next half block, one iteration ahead
      const BlockGeom& G = a.geom[t_next >> 1];
      s.invd[phase ^ 1][0] = G.invD[0]; s.invd[phase ^ 1][1] = G.invD[1]; s.invd[phase ^ 1][2] = G.invD[2];
    }
    mbar_wait(&s.mbar_tile, phase);

    // ---- O-3: conserved -> primitive, in place
    {
      double rho, p, me[4];
      to_primitive<MV>(&s.M[0][0] + g_off, a.gm1, rho, p, me);
      if (tid < NPH) {
        to_primitive<ZV>((tid < ZV ? &s.ZM[0][0] : &s.ZP[0][0]) + (tid & (ZV - 1)), a.gm1, rho, p, me);
        double* q = &s.M[0][0] + m_off(i, j, kk);
        to_primitive<MV>(q, a.gm1, rho, p, me);
        if (STAGE == 1) {                                // stage 1: U^n is the stage input itself
          U[0] = rho; U[1] = me[0]; U[2] = me[1]; U[3] = me[2];
          U[4] = q[4 * MV]; U[5] = q[5 * MV]; U[6] = q[6 * MV]; U[7] = me[3];
        }
        int warn = 0;
        if (!isfinite(rho) || !isfinite(p)) warn |= BATL_WARN_NONFINITE;
        if (rho <= 0.0 || p <= 0.0) warn |= BATL_WARN_NEGATIVE;
        if (warn) atomicOr(&a.sc->warn, warn);
      }
    }
    __syncthreads();

    const double* geo = s.invd[phase];
    SweepAcc acc;
    acc.divb = 0.0; acc.speed = 0.0;
    auto nothing = [] {};
    constexpr bool ACC = STAGE != 0;
    sweep<0, ACC, BETA2>(s, tid, i, j, kk, a.half_beta, a.gamma, a.inv_gm1, geo, a.use_divb, U, acc, nothing);
    sweep<1, ACC, BETA2>(s, tid, i, j, kk, a.half_beta, a.gamma, a.inv_gm1, geo, a.use_divb, U, acc, nothing);
    sweep<2, ACC, BETA2>(s, tid, i, j, kk, a.half_beta, a.gamma, a.inv_gm1, geo, a.use_divb, U, acc, [&] {
      if (tid == 0 && t_next < n_tiles) {                // the tile is dead: fetch the next one
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        request_tile(s, maps, t_next);
      }
    });

    if (tid < NPH) {
      if (STAGE != 1) dt_min = dmin(dt_min, a.cfl * fast_rcp(acc.speed));    // O-8
      if (STAGE != 0) {
#pragma unroll
        for (int v = 0; v < NV; ++v) a.out[g0 + (size_t)v * NCELL] = U[v];   // O-7
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

struct MapCacheEntry { const double* base; int n_blocks; TileMaps maps; };
std::mutex g_cache_mutex;
std::vector<MapCacheEntry> g_cache;

bool get_maps(const double* base, int n_blocks, TileMaps* out) {
  std::lock_guard<std::mutex> lock(g_cache_mutex);
  for (const auto& e : g_cache)
    if (e.base == base && e.n_blocks == n_blocks) { *out = e.maps; return true; }
  MapCacheEntry e;
  e.base = base; e.n_blocks = n_blocks;
  if (!make_map(&e.maps.m, base, n_blocks, NS, NS, HK)) return false;
  if (!make_map(&e.maps.z, base, n_blocks, NI, NI, NG)) return false;
  if (g_cache.size() >= 64) g_cache.erase(g_cache.begin());
  g_cache.push_back(e);
  *out = e.maps;
  return true;
}

}  // namespace

// local time stepping scales the update of a cell by its own dt_c, which is only known after
// all three sweeps; those runs (and B0 / body blocks) take the general kernel
bool stage_fused_supports(const StageArgs& a) {
  return a.use_b0 == 0 && a.use_body == 0 && a.dt_mode != BATL_DT_LOCAL;
}

template <int STAGE, bool BETA2>
cudaError_t set_smem_attribute() {
  return cudaFuncSetAttribute(stage_fused_kernel<STAGE, BETA2>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                              (int)sizeof(FusedSmem));
}

cudaError_t init_fused_attributes() {
  cudaError_t e;
  if ((e = set_smem_attribute<0, false>()) != cudaSuccess) return e;
  if ((e = set_smem_attribute<1, false>()) != cudaSuccess) return e;
  if ((e = set_smem_attribute<2, false>()) != cudaSuccess) return e;
  if ((e = set_smem_attribute<0, true>()) != cudaSuccess) return e;
  if ((e = set_smem_attribute<1, true>()) != cudaSuccess) return e;
  return set_smem_attribute<2, true>();
}

cudaError_t launch_stage_fused(int stage, const StageArgs& a, cudaStream_t st) {
  if (a.n_blocks == 0) return cudaSuccess;
  TileMaps maps;
  if (!get_maps(a.in, a.n_blocks, &maps)) return cudaErrorNotSupported;
  static int n_sm = 0;
  if (n_sm == 0) {
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
  }
  const int n_tiles = 2 * a.n_blocks;                      // half blocks
  const int grid = n_tiles < 2 * n_sm ? n_tiles : 2 * n_sm; // persistent: two CTAs per SM
  const size_t sm = sizeof(FusedSmem);
  if (a.beta == 2.0) {                                     // compile-time special case of the default limiter
    if (stage == 0) stage_fused_kernel<0, true><<<grid, FT, sm, st>>>(maps, a, n_tiles);
    else if (stage == 1) stage_fused_kernel<1, true><<<grid, FT, sm, st>>>(maps, a, n_tiles);
    else stage_fused_kernel<2, true><<<grid, FT, sm, st>>>(maps, a, n_tiles);
  } else {
    if (stage == 0) stage_fused_kernel<0, false><<<grid, FT, sm, st>>>(maps, a, n_tiles);
    else if (stage == 1) stage_fused_kernel<1, false><<<grid, FT, sm, st>>>(maps, a, n_tiles);
    else stage_fused_kernel<2, false><<<grid, FT, sm, st>>>(maps, a, n_tiles);
  }
  return cudaGetLastError();
}

}  // namespace batl
