// Fused stage kernel (steps a5-a9) for blocks without B0 split and without body cells:
// reconstruction + Rusanov flux + 8-wave source + update + dt minimum in one pass,
// face states and fluxes never leave the SM (the paper's GPU code passes them through
// global Flux_V[XYZ]B arrays, Alg. 2 L76, L82-84).
//
// Work decomposition (sm_100a, 148 SMs, 228 KB shared memory per SM):
//   * the unit of work is a HALF block: 8 x 8 x 4 physical cells plus the face ghost
//     slabs they need (768 cells x 8 variables = 48 KB).  The kernel is persistent: two
//     CTAs per SM, each walking the half blocks t = blockIdx.x, blockIdx.x + gridDim.x, ...
//   * software pipeline: the tile of the NEXT half block is requested as soon as the last
//     slope of the current one has been taken (middle of the z sweep), so its HBM latency
//     hides behind the z fluxes, the update and the stores; U^n of the physical cells
//     (the `base` of stage 2) arrives by TMA in a buffer of its own, one half block ahead.
//     In stage 1 base = input, so it is saved from the tile and never re-read from HBM.
//   * the tile is fetched by TMA tensor copies (cp.async.bulk.tensor.4d -> UTMALDG) into
//     a layout that is dense per slab: rows of 8 doubles, no 12-wide rows, hence no
//     shared-memory bank conflicts on the row-contiguous accesses.  Edge and corner
//     ghost rows are never read.
//   * 256 "cell" threads own one physical cell each for all three sweeps (accumulators
//     stay in registers); 64 "helper" threads do the slopes of the ghost cells next to
//     the block faces and the fluxes of the low boundary faces.
//   * per sweep: every cell computes ONE limited slope per variable, keeps W^L of its
//     high face in registers and hands W^R of its low face to the neighbour through
//     shared memory; the flux of a face is computed once, by the thread left of it.
#include <cuda.h>

#include <mutex>
#include <vector>

#include "batl_device.cuh"
#include "mhd_physics.cuh"

namespace batl {
namespace {

constexpr int FT = 320;                 // threads per CTA: 256 cell threads + 64 helpers
constexpr int HK = 4;                   // physical k planes per CTA
constexpr int TILE = 768;               // cells per variable in the shared-memory tile
constexpr int OFF_GXM = 256, OFF_GXP = 320, OFF_GYM = 384, OFF_GYP = 448, OFF_GZM = 512, OFF_GZP = 640;
constexpr int NSLOT = 320;              // face slots per sweep: 256 high faces + up to 64 low boundary faces
constexpr uint32_t TILE_BYTES = TILE * NV * sizeof(double);   // 49,152

constexpr int NPH = 256;                // physical cells of a half block
constexpr uint32_t BASE_BYTES = NPH * NV * sizeof(double);    // 16,384

struct FusedSmem {
  double tile[NV][TILE];                // primitives after the in-place conversion
  double wr[NV][NSLOT];                 // W^R of the face in slot s
  double fx[NV + 2][NSLOT];             // 2*flux, B_n, c_max of the face in slot s
  double base[NV][NPH];                 // U^n of the physical cells (conserved)
  double xl[NSLOT];                     // z sweep: B_z of W^L of the face in slot s (early div B)
  double invd[2][4];                    // 1 / D_d of the current and of the next half block
  double red[8];
  unsigned long long mbar_tile, mbar_base;
};

struct TileMaps { CUtensorMap p, gx, gy, gz; };

__device__ __forceinline__ void mbar_wait(unsigned long long* mbar, uint32_t parity) {
  uint32_t done = 0;
  while (!done) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done) : "r"((uint32_t)__cvta_generic_to_shared(mbar)), "r"(parity) : "memory");
  }
}

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void tma_load_4d(void* dst, const CUtensorMap* map, unsigned long long* mbar,
                                            int c0, int c1, int c2, int c3) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
      ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(mbar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
      : "memory");
}

// offset of cell (i, j, kk) inside one variable of the tile; at most one coordinate is a ghost
__device__ __forceinline__ int cell_off(int i, int j, int kk) {
  if (i < 0) return OFF_GXM + (kk * 8 + j) * 2 + (i + 2);
  if (i >= NI) return OFF_GXP + (kk * 8 + j) * 2 + (i - NI);
  if (j < 0) return OFF_GYM + (kk * 2 + (j + 2)) * 8 + i;
  if (j >= NI) return OFF_GYP + (kk * 2 + (j - NI)) * 8 + i;
  if (kk < 0) return OFF_GZM + ((kk + 2) * 8 + j) * 8 + i;
  if (kk >= HK) return OFF_GZP + ((kk - HK) * 8 + j) * 8 + i;
  return (kk * 8 + j) * 8 + i;
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

__device__ __forceinline__ double half_slope(double dm, double dp, double hb) {
  // |.| only ever appears as an operand modifier, so no instruction is spent on it
  const double sel = (fabs(dm) < fabs(dp)) ? dm : dp;
  const double lim = dmin(hb * fabs(sel), 0.25 * (fabs(dm) + fabs(dp)));
  const int hi_dm = __double2hiint(dm);
  const bool opposite = (hi_dm ^ __double2hiint(dp)) < 0;
  // copysign(lim, dm): lim >= 0, so OR-ing the sign bit of dm is enough
  const double h = __hiloint2double(__double2hiint(lim) | (hi_dm & 0x80000000), __double2loint(lim));
  return opposite ? 0.0 : h;
}

// slopes of one cell in direction D: W^L of its high face, W^R of its low face; W0 = the cell itself
__device__ __forceinline__ void cell_faces(const double* __restrict__ tile, int cm, int c0, int cp, double hb,
                                           double WL[NV], double WR[NV], double W0[NV]) {
#pragma unroll
  for (int v = 0; v < NV; ++v) {
    const double w0 = tile[v * TILE + c0];
    const double h = half_slope(w0 - tile[v * TILE + cm], tile[v * TILE + cp] - w0, hb);
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

// per-thread running sums of a half block; the state itself is accumulated in shared memory:
// s.base starts as U^n and receives f dt (-dF_d / D_d + S) sweep by sweep, so no accumulator
// registers live across the flux evaluations (they used to spill).
struct SweepAcc { double divb; double speed; };

// One direction sweep of the half block (see the header comment).  hinv = 1 / (2 D_d).
// The z sweep (D = 2) is the last one: once its slopes are taken the tile is dead, `tile_dead`
// runs right after the barrier (it requests the next tile), and the 8-wave source (O-6) is
// applied there, while the cell-centre u and B1 are still in registers -- the B_n of the two
// z faces is already known from the face states, ahead of their fluxes.
template <int D, bool ACCUM, class Hook, class Hook2>
__device__ __forceinline__ void sweep(FusedSmem& s, int tid, int i, int j, int kk, double hb, double gamma,
                                      double inv_gm1, double hinv, double invd, double f, int use_divb, SweepAcc& acc,
                                      Hook&& tile_dead, Hook2&& before_accumulate) {
  constexpr int NB = (D == 2) ? 64 : 32;               // low boundary faces of the half block
  const double* __restrict__ tile = &s.tile[0][0];
  double* __restrict__ wr = &s.wr[0][0];
  double* __restrict__ fx = &s.fx[0][0];
  double WL[NV], WR[NV], W0[NV];
  int slot_minus = 0;
  if (tid < 256) {
    const int cm = cell_off(i - (D == 0), j - (D == 1), kk - (D == 2));
    const int cp = cell_off(i + (D == 0), j + (D == 1), kk + (D == 2));
    const int pos = (D == 0) ? i : (D == 1) ? j : kk;
    const int bidx = (D == 0) ? (tid >> 3) : (D == 1) ? (i + 8 * kk) : (i + 8 * j);
    constexpr int stride = (D == 0) ? 1 : (D == 1) ? 8 : 64;
    slot_minus = (pos > 0) ? tid - stride : 256 + bidx;
    cell_faces(tile, cm, tid, cp, hb, WL, WR, W0);
#pragma unroll
    for (int v = 0; v < NV; ++v) wr[v * NSLOT + slot_minus] = WR[v];
    if (D == 2) s.xl[tid] = WL[6];
  } else {
    const int p = tid - 256;
    double dummy[NV];
    if (p < NB) {                                      // ghost cell below the low face: its W^L
      const int a = p & 7, b = p >> 3;
      const int gi = (D == 0) ? -1 : a, gj = (D == 1) ? -1 : (D == 0 ? a : b), gk = (D == 2) ? -1 : b;
      const int cm = cell_off(gi - (D == 0), gj - (D == 1), gk - (D == 2));
      const int c0 = cell_off(gi, gj, gk);
      const int cp = cell_off(gi + (D == 0), gj + (D == 1), gk + (D == 2));
      cell_faces(tile, cm, c0, cp, hb, WL, dummy, W0);
      if (D == 2) s.xl[tid] = WL[6];
    }
    const int q = (D == 2) ? p : p - 32;               // ghost cell above the high face: its W^R
    if (q >= 0) {
      const int a = q & 7, b = q >> 3;
      const int top = (D == 2) ? HK : NI;
      const int gi = (D == 0) ? top : a, gj = (D == 1) ? top : (D == 0 ? a : b), gk = (D == 2) ? top : b;
      const int cm = cell_off(gi - (D == 0), gj - (D == 1), gk - (D == 2));
      const int c0 = cell_off(gi, gj, gk);
      const int cp = cell_off(gi + (D == 0), gj + (D == 1), gk + (D == 2));
      cell_faces(tile, cm, c0, cp, hb, dummy, WR, W0);
      const int slot = cm;                             // the last physical cell owns the slot of that face
#pragma unroll
      for (int v = 0; v < NV; ++v) wr[v * NSLOT + slot] = WR[v];
    }
  }
  __syncthreads();
  tile_dead();
  if (tid < 256 + NB) {
    double F2[NV], Bn2, c;
    const double wr_own_bn = WR[6];
#pragma unroll
    for (int v = 0; v < NV; ++v) WR[v] = wr[v * NSLOT + tid];
    if (D == 2 && tid < 256 && use_divb) {             // O-6: 8-wave source, cell-centre state of the stage input
      const double d = -f * fma((WL[6] + WR[6]) - (s.xl[slot_minus] + wr_own_bn), hinv, acc.divb);
      const double ub = W0[1] * W0[4] + W0[2] * W0[5] + W0[3] * W0[6];
      if (ACCUM) {
#pragma unroll
        for (int q = 0; q < 3; ++q) {
          s.base[1 + q][tid] = fma(W0[4 + q], d, s.base[1 + q][tid]);
          s.base[4 + q][tid] = fma(W0[1 + q], d, s.base[4 + q][tid]);
        }
        s.base[7][tid] = fma(ub, d, s.base[7][tid]);
      }
    }
    face_flux2<D>(WL, WR, gamma, inv_gm1, F2, Bn2, c);
#pragma unroll
    for (int v = 0; v < NV; ++v) fx[v * NSLOT + tid] = F2[v];
    if (D != 2) fx[NV * NSLOT + tid] = Bn2;
    fx[(NV + 1) * NSLOT + tid] = c;
  }
  __syncthreads();
  before_accumulate();
  if (tid < 256) {
    // both faces of the cell are read back from shared memory (the own one too: keeping it in
    // registers across the barrier made the compiler spill)
    if (ACCUM) {
      const double fh = f * hinv;
#pragma unroll
      for (int v = 0; v < NV; ++v)
        s.base[v][tid] = fma(fx[v * NSLOT + slot_minus] - fx[v * NSLOT + tid], fh, s.base[v][tid]);
    }
    if (D != 2) acc.divb = fma(fx[NV * NSLOT + tid] - fx[NV * NSLOT + slot_minus], hinv, acc.divb);
    acc.speed = fma(dmax(fx[(NV + 1) * NSLOT + tid], fx[(NV + 1) * NSLOT + slot_minus]), invd, acc.speed);
  }
}

// TMA requests of one half block; issued by lane 0 of warps 0..7, one variable each
__device__ __forceinline__ void request_tile(FusedSmem& s, const TileMaps& maps, int t, int v) {
  const int b = t >> 1, k0 = NG + HK * (t & 1);
  const int c3 = b * NV + v;
  double* dst = &s.tile[v][0];
  tma_load_4d(dst, &maps.p, &s.mbar_tile, NG, NG, k0, c3);
  tma_load_4d(dst + OFF_GXM, &maps.gx, &s.mbar_tile, 0, NG, k0, c3);
  tma_load_4d(dst + OFF_GXP, &maps.gx, &s.mbar_tile, NG + NI, NG, k0, c3);
  tma_load_4d(dst + OFF_GYM, &maps.gy, &s.mbar_tile, NG, 0, k0, c3);
  tma_load_4d(dst + OFF_GYP, &maps.gy, &s.mbar_tile, NG, NG + NI, k0, c3);
  tma_load_4d(dst + OFF_GZM, &maps.gz, &s.mbar_tile, NG, NG, k0 - NG, c3);
  tma_load_4d(dst + OFF_GZP, &maps.gz, &s.mbar_tile, NG, NG, k0 + HK, c3);
}

template <int STAGE>
__global__ void __launch_bounds__(FT, 2)
stage_fused_kernel(const __grid_constant__ TileMaps maps, const __grid_constant__ CUtensorMap base_map,
                   const StageArgs a, const int n_tiles) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  FusedSmem& s = *reinterpret_cast<FusedSmem*>(smem_raw);
  const int tid = threadIdx.x;
  const bool issuer = (tid & 31) == 0 && tid < 256;     // lane 0 of warp v moves variable v
  const int stride = gridDim.x;
  int t = blockIdx.x;

  if (tid == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(&s.mbar_tile)));
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(&s.mbar_base)));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (tid == 32 && t < n_tiles) {                       // 1 / D_d of the first half block
    const BlockGeom& G = a.geom[t >> 1];
    s.invd[0][0] = G.invD[0]; s.invd[0][1] = G.invD[1]; s.invd[0][2] = G.invD[2];
  }
  __syncthreads();
  if (t < n_tiles) {
    if (tid == 0) {
      asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(&s.mbar_tile)), "r"(TILE_BYTES) : "memory");
      if (STAGE == 2)
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(&s.mbar_base)), "r"(BASE_BYTES) : "memory");
    }
    if (issuer) {
      request_tile(s, maps, t, tid >> 5);
      if (STAGE == 2)
        tma_load_4d(&s.base[tid >> 5][0], &base_map, &s.mbar_base, NG, NG, NG + HK * (t & 1), (t >> 1) * NV + (tid >> 5));
    }
  }

  const int i = tid & 7, j = (tid >> 3) & 7, kk = (tid >> 6) & 3;
  // O-7: U = U^n + f R with f = dt/2 (stage 1) or dt (stage 2); dt is global or fixed here
  const double f = (STAGE == 0) ? 0.0 : (STAGE == 1 ? 0.5 : 1.0) * a.sc->dt;
  const double INF = __longlong_as_double(0x7FF0000000000000ll);
  double dt_min = INF;
  int warn = 0;
  uint32_t phase = 0;

  for (; t < n_tiles; t += stride, phase ^= 1) {
    const int b = t >> 1;
    const int k0 = NG + HK * (t & 1);                    // first physical storage plane of this half
    const int t_next = t + stride;
    if (tid == 32 && t_next < n_tiles) {                 // geometry of the next half block, one iteration ahead
      const BlockGeom& G = a.geom[t_next >> 1];
      s.invd[phase ^ 1][0] = G.invD[0]; s.invd[phase ^ 1][1] = G.invD[1]; s.invd[phase ^ 1][2] = G.invD[2];
    }
    mbar_wait(&s.mbar_tile, phase);

    // ---- O-3: conserved -> primitive, in place; stage 1 keeps U^n of the physical cells
    for (int c = tid; c < TILE; c += FT) {
      const double rho = s.tile[0][c];
      const double ir = fast_rcp(rho);
      const double mx = s.tile[1][c], my = s.tile[2][c], mz = s.tile[3][c], e = s.tile[7][c];
      const double ux = mx * ir, uy = my * ir, uz = mz * ir;
      const double bx = s.tile[4][c], by = s.tile[5][c], bz = s.tile[6][c];
      const double ke = 0.5 * rho * (ux * ux + uy * uy + uz * uz);
      const double me = 0.5 * (bx * bx + by * by + bz * bz);
      const double p = a.gm1 * (e - ke - me);
      s.tile[1][c] = ux; s.tile[2][c] = uy; s.tile[3][c] = uz; s.tile[7][c] = p;
      if (c < NPH) {
        if (STAGE == 1) {
          s.base[0][c] = rho; s.base[1][c] = mx; s.base[2][c] = my; s.base[3][c] = mz;
          s.base[4][c] = bx; s.base[5][c] = by; s.base[6][c] = bz; s.base[7][c] = e;
        }
        if (!isfinite(rho) || !isfinite(p)) warn |= BATL_WARN_NONFINITE;
        if (rho <= 0.0 || p <= 0.0) warn |= BATL_WARN_NEGATIVE;
      }
    }
    __syncthreads();

    const double idx = s.invd[phase][0], idy = s.invd[phase][1], idz = s.invd[phase][2];
    SweepAcc acc;
    acc.divb = 0.0; acc.speed = 0.0;
    auto nothing = [] {};
    constexpr bool ACC = STAGE != 0;
    sweep<0, ACC>(s, tid, i, j, kk, a.half_beta, a.gamma, a.inv_gm1, 0.5 * idx, idx, f, a.use_divb, acc, nothing,
                  [&] { if (STAGE == 2) mbar_wait(&s.mbar_base, phase); });
    sweep<1, ACC>(s, tid, i, j, kk, a.half_beta, a.gamma, a.inv_gm1, 0.5 * idy, idy, f, a.use_divb, acc, nothing, nothing);
    sweep<2, ACC>(s, tid, i, j, kk, a.half_beta, a.gamma, a.inv_gm1, 0.5 * idz, idz, f, a.use_divb, acc, [&] {
      if (t_next < n_tiles) {                            // the tile is dead: fetch the next one
        if (tid == 0)
          asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(&s.mbar_tile)), "r"(TILE_BYTES) : "memory");
        if (issuer) {
          asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
          request_tile(s, maps, t_next, tid >> 5);
        }
      }
    }, nothing);

    if (tid < NPH) {
      if (STAGE != 1) dt_min = dmin(dt_min, a.cfl * fast_rcp(acc.speed));    // O-8
      if (STAGE != 0) {
        const size_t g0 = (size_t)b * BLOCK_DOUBLES + ((size_t)(k0 + kk) * NS + (j + NG)) * NS + (i + NG);
#pragma unroll
        for (int v = 0; v < NV; ++v) a.out[g0 + (size_t)v * NCELL] = s.base[v][tid];   // O-7, summed in place
      }
    }
    __syncthreads();                                      // base, wr and fx are free again
    if (STAGE == 2 && t_next < n_tiles) {
      if (tid == 0)
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(&s.mbar_base)), "r"(BASE_BYTES) : "memory");
      if (issuer) {
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        tma_load_4d(&s.base[tid >> 5][0], &base_map, &s.mbar_base, NG, NG, NG + HK * (t_next & 1),
                    (t_next >> 1) * NV + (tid >> 5));
      }
    }
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
  if (warn) atomicOr(&a.sc->warn, warn);
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

bool make_map(CUtensorMap* m, const double* base, int n_blocks, int bi, int bj, int bk) {
  EncodeTiledFn enc = encode_fn();
  if (!enc) return false;
  const cuuint64_t dims[4] = {NS, NS, NS, (cuuint64_t)n_blocks * NV};
  const cuuint64_t strides[3] = {NS * sizeof(double), NS * NS * sizeof(double), NCELL * sizeof(double)};
  const cuuint32_t box[4] = {(cuuint32_t)bi, (cuuint32_t)bj, (cuuint32_t)bk, 1};
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
  if (!make_map(&e.maps.p, base, n_blocks, NI, NI, HK)) return false;
  if (!make_map(&e.maps.gx, base, n_blocks, NG, NI, HK)) return false;
  if (!make_map(&e.maps.gy, base, n_blocks, NI, NG, HK)) return false;
  if (!make_map(&e.maps.gz, base, n_blocks, NI, NI, NG)) return false;
  if (g_cache.size() >= 64) g_cache.erase(g_cache.begin());
  g_cache.push_back(e);
  *out = e.maps;
  return true;
}

}  // namespace

// local time stepping needs dt_c of the cell before the update can be scaled, which the in-place
// accumulation above cannot provide; those runs (and B0 / body blocks) take the general kernel
bool stage_fused_supports(const StageArgs& a) {
  return a.use_b0 == 0 && a.use_body == 0 && a.dt_mode != BATL_DT_LOCAL;
}

cudaError_t init_fused_attributes() {
  cudaError_t e;
  e = cudaFuncSetAttribute(stage_fused_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(FusedSmem));
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(stage_fused_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(FusedSmem));
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(stage_fused_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(FusedSmem));
}

cudaError_t launch_stage_fused(int stage, const StageArgs& a, cudaStream_t st) {
  if (a.n_blocks == 0) return cudaSuccess;
  TileMaps maps, base_maps;
  if (!get_maps(a.in, a.n_blocks, &maps)) return cudaErrorNotSupported;
  if (!get_maps(a.base, a.n_blocks, &base_maps)) return cudaErrorNotSupported;
  static int n_sm = 0;
  if (n_sm == 0) {
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
  }
  const int n_tiles = 2 * a.n_blocks;                      // half blocks
  const int grid = n_tiles < 2 * n_sm ? n_tiles : 2 * n_sm; // persistent: two CTAs per SM
  const size_t sm = sizeof(FusedSmem);
  if (stage == 0) stage_fused_kernel<0><<<grid, FT, sm, st>>>(maps, base_maps.p, a, n_tiles);
  else if (stage == 1) stage_fused_kernel<1><<<grid, FT, sm, st>>>(maps, base_maps.p, a, n_tiles);
  else stage_fused_kernel<2><<<grid, FT, sm, st>>>(maps, base_maps.p, a, n_tiles);
  return cudaGetLastError();
}

}  // namespace batl
