// Fused stage kernel (steps a5-a9) for blocks without B0 split and without body cells:
// reconstruction + Rusanov flux + 8-wave source + update + dt minimum in one pass,
// face states and fluxes never leave the SM (the paper's GPU code passes them through
// global Flux_V[XYZ]B arrays, Alg. 2 L76, L82-84).
//
// Work decomposition (sm_100a, 148 SMs, 228 KB shared memory per SM):
//   * one CTA per HALF block: 8 x 8 x 4 physical cells plus the face ghost slabs they
//     need (768 cells x 8 variables = 48 KB).  Two CTAs fit on one SM, so the TMA load
//     of one overlaps the arithmetic of the other.
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

struct FusedSmem {
  double tile[NV][TILE];                // primitives after the in-place conversion
  double wr[NV][NSLOT];                 // W^R of the face in slot s
  double fx[NV + 2][NSLOT];             // 2*flux, B_n, c_max of the face in slot s
  double red[8];
  unsigned long long mbar;
};

struct TileMaps { CUtensorMap p, gx, gy, gz; };

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

// slopes of one cell in direction D: W^L of its high face, W^R of its low face
__device__ __forceinline__ void cell_faces(const double* __restrict__ tile, int cm, int c0, int cp, double hb,
                                           double WL[NV], double WR[NV]) {
#pragma unroll
  for (int v = 0; v < NV; ++v) {
    const double w0 = tile[v * TILE + c0];
    const double h = half_slope(w0 - tile[v * TILE + cm], tile[v * TILE + cp] - w0, hb);
    WL[v] = w0 + h;
    WR[v] = w0 - h;
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

struct SweepAcc { double R[NV]; double divb; double speed; };

// One direction sweep of the half block (see the header comment).  hinv = 1 / (2 D_d).
template <int D>
__device__ __forceinline__ void sweep(FusedSmem& s, int tid, int i, int j, int kk, double hb, double gamma,
                                      double inv_gm1, double hinv, double invd, SweepAcc& acc) {
  constexpr int NB = (D == 2) ? 64 : 32;               // low boundary faces of the half block
  const double* __restrict__ tile = &s.tile[0][0];
  double* __restrict__ wr = &s.wr[0][0];
  double* __restrict__ fx = &s.fx[0][0];
  double WL[NV], WR[NV];
  int slot_minus = 0;
  if (tid < 256) {
    const int cm = cell_off(i - (D == 0), j - (D == 1), kk - (D == 2));
    const int cp = cell_off(i + (D == 0), j + (D == 1), kk + (D == 2));
    const int pos = (D == 0) ? i : (D == 1) ? j : kk;
    const int bidx = (D == 0) ? (tid >> 3) : (D == 1) ? (i + 8 * kk) : (i + 8 * j);
    constexpr int stride = (D == 0) ? 1 : (D == 1) ? 8 : 64;
    slot_minus = (pos > 0) ? tid - stride : 256 + bidx;
    cell_faces(tile, cm, tid, cp, hb, WL, WR);
#pragma unroll
    for (int v = 0; v < NV; ++v) wr[v * NSLOT + slot_minus] = WR[v];
  } else {
    const int p = tid - 256;
    if (p < NB) {                                      // ghost cell below the low face: its W^L
      const int a = p & 7, b = p >> 3;
      const int gi = (D == 0) ? -1 : a, gj = (D == 1) ? -1 : (D == 0 ? a : b), gk = (D == 2) ? -1 : b;
      const int cm = cell_off(gi - (D == 0), gj - (D == 1), gk - (D == 2));
      const int c0 = cell_off(gi, gj, gk);
      const int cp = cell_off(gi + (D == 0), gj + (D == 1), gk + (D == 2));
      double dummy[NV];
      cell_faces(tile, cm, c0, cp, hb, WL, dummy);
    }
    const int q = (D == 2) ? p : p - 32;               // ghost cell above the high face: its W^R
    if (q >= 0) {
      const int a = q & 7, b = q >> 3;
      const int top = (D == 2) ? HK : NI;
      const int gi = (D == 0) ? top : a, gj = (D == 1) ? top : (D == 0 ? a : b), gk = (D == 2) ? top : b;
      const int cm = cell_off(gi - (D == 0), gj - (D == 1), gk - (D == 2));
      const int c0 = cell_off(gi, gj, gk);
      const int cp = cell_off(gi + (D == 0), gj + (D == 1), gk + (D == 2));
      double dummy[NV];
      cell_faces(tile, cm, c0, cp, hb, dummy, WR);
      const int slot = cm;                             // the last physical cell owns the slot of that face
#pragma unroll
      for (int v = 0; v < NV; ++v) wr[v * NSLOT + slot] = WR[v];
    }
  }
  __syncthreads();
  double F2[NV], Bn2 = 0.0, c = 0.0;
  if (tid < 256 + NB) {
#pragma unroll
    for (int v = 0; v < NV; ++v) WR[v] = wr[v * NSLOT + tid];
    face_flux2<D>(WL, WR, gamma, inv_gm1, F2, Bn2, c);
#pragma unroll
    for (int v = 0; v < NV; ++v) fx[v * NSLOT + tid] = F2[v];
    fx[NV * NSLOT + tid] = Bn2;
    fx[(NV + 1) * NSLOT + tid] = c;
  }
  __syncthreads();
  if (tid < 256) {
#pragma unroll
    for (int v = 0; v < NV; ++v) acc.R[v] = fma(fx[v * NSLOT + slot_minus] - F2[v], hinv, acc.R[v]);
    acc.divb = fma(Bn2 - fx[NV * NSLOT + slot_minus], hinv, acc.divb);
    acc.speed = fma(dmax(c, fx[(NV + 1) * NSLOT + slot_minus]), invd, acc.speed);
  }
}

template <int STAGE>
__global__ void __launch_bounds__(FT, 2)
stage_fused_kernel(const __grid_constant__ TileMaps maps, const StageArgs a) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  FusedSmem& s = *reinterpret_cast<FusedSmem*>(smem_raw);
  const int tid = threadIdx.x;
  const int b = blockIdx.x >> 1, half = blockIdx.x & 1;
  const int k0 = NG + HK * half;                        // first physical storage plane of this half

  if (tid == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(&s.mbar)));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  if (tid == 0)
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(&s.mbar)), "r"(TILE_BYTES) : "memory");
  if ((tid & 31) == 0 && tid < 256) {                   // lane 0 of warp v fetches variable v
    const int v = tid >> 5;
    const int c3 = b * NV + v;
    double* dst = &s.tile[v][0];
    tma_load_4d(dst, &maps.p, &s.mbar, NG, NG, k0, c3);
    tma_load_4d(dst + OFF_GXM, &maps.gx, &s.mbar, 0, NG, k0, c3);
    tma_load_4d(dst + OFF_GXP, &maps.gx, &s.mbar, NG + NI, NG, k0, c3);
    tma_load_4d(dst + OFF_GYM, &maps.gy, &s.mbar, NG, 0, k0, c3);
    tma_load_4d(dst + OFF_GYP, &maps.gy, &s.mbar, NG, NG + NI, k0, c3);
    tma_load_4d(dst + OFF_GZM, &maps.gz, &s.mbar, NG, NG, k0 - NG, c3);
    tma_load_4d(dst + OFF_GZP, &maps.gz, &s.mbar, NG, NG, k0 + HK, c3);
  }

  const BlockGeom G = a.geom[b];
  const double gm1 = a.gamma - 1.0, inv_gm1 = 1.0 / gm1, hb = 0.5 * a.beta;
  const int i = tid & 7, j = (tid >> 3) & 7, kk = (tid >> 6) & 3;

  {                                                      // wait for the tile
    uint32_t done = 0;
    while (!done) {
      asm volatile(
          "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
          : "=r"(done) : "r"(smem_u32(&s.mbar)), "r"(0u) : "memory");
    }
  }

  // ---- O-3: conserved -> primitive, in place
  int warn = 0;
  for (int c = tid; c < TILE; c += FT) {
    const double rho = s.tile[0][c];
    const double ir = fast_rcp(rho);
    const double ux = s.tile[1][c] * ir, uy = s.tile[2][c] * ir, uz = s.tile[3][c] * ir;
    const double bx = s.tile[4][c], by = s.tile[5][c], bz = s.tile[6][c];
    const double ke = 0.5 * rho * (ux * ux + uy * uy + uz * uz);
    const double me = 0.5 * (bx * bx + by * by + bz * bz);
    const double p = gm1 * (s.tile[7][c] - ke - me);
    s.tile[1][c] = ux; s.tile[2][c] = uy; s.tile[3][c] = uz; s.tile[7][c] = p;
    if (c < 256) {
      if (!isfinite(rho) || !isfinite(p)) warn |= BATL_WARN_NONFINITE;
      if (rho <= 0.0 || p <= 0.0) warn |= BATL_WARN_NEGATIVE;
    }
  }
  __syncthreads();

  SweepAcc acc;
#pragma unroll
  for (int v = 0; v < NV; ++v) acc.R[v] = 0.0;
  acc.divb = 0.0; acc.speed = 0.0;
  sweep<0>(s, tid, i, j, kk, hb, a.gamma, inv_gm1, 0.5 * G.invD[0], G.invD[0], acc);
  sweep<1>(s, tid, i, j, kk, hb, a.gamma, inv_gm1, 0.5 * G.invD[1], G.invD[1], acc);
  sweep<2>(s, tid, i, j, kk, hb, a.gamma, inv_gm1, 0.5 * G.invD[2], G.invD[2], acc);

  double dt_c = __longlong_as_double(0x7FF0000000000000ll);
  if (tid < 256) {
    // ---- O-6: 8-wave source from the cell-centre state
    if (a.use_divb) {
      const double ux = s.tile[1][tid], uy = s.tile[2][tid], uz = s.tile[3][tid];
      const double bx = s.tile[4][tid], by = s.tile[5][tid], bz = s.tile[6][tid];
      const double d = acc.divb;
      acc.R[1] = fma(-bx, d, acc.R[1]); acc.R[2] = fma(-by, d, acc.R[2]); acc.R[3] = fma(-bz, d, acc.R[3]);
      acc.R[4] = fma(-ux, d, acc.R[4]); acc.R[5] = fma(-uy, d, acc.R[5]); acc.R[6] = fma(-uz, d, acc.R[6]);
      acc.R[7] = fma(-(ux * bx + uy * by + uz * bz), d, acc.R[7]);
    }
    dt_c = a.cfl * fast_rcp(acc.speed);                 // O-8
    if (STAGE != 0) {
      const int cell = tid + 256 * half;                // physical cell index in the block
      double dt;
      if (a.dt_mode == BATL_DT_LOCAL) {                 // Q-T3
        double* dtl = a.dt_local + (size_t)b * NPHYS + cell;
        if (STAGE == 1) *dtl = dt_c;
        dt = (STAGE == 1) ? dt_c : *dtl;
      } else {
        dt = a.sc->dt;
      }
      const double f = (STAGE == 1 ? 0.5 : 1.0) * dt;
      const size_t g0 = (size_t)b * BLOCK_DOUBLES + ((size_t)(k0 + kk) * NS + (j + NG)) * NS + (i + NG);
#pragma unroll
      for (int v = 0; v < NV; ++v)                      // O-7
        a.out[g0 + (size_t)v * NCELL] = fma(f, acc.R[v], a.base[g0 + (size_t)v * NCELL]);
    }
  }

  // ---- a9: minimum of dt_c over the CTA, one atomic
  if (STAGE != 1 && a.dt_mode == BATL_DT_GLOBAL) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) dt_c = fmin(dt_c, __shfl_xor_sync(0xffffffffu, dt_c, o));
    if ((tid & 31) == 0 && tid < 256) s.red[tid >> 5] = dt_c;
    __syncthreads();
    if (tid < 32) {
      double v = (tid < 8) ? s.red[tid] : __longlong_as_double(0x7FF0000000000000ll);
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

bool stage_fused_supports(const StageArgs& a) { return a.use_b0 == 0 && a.use_body == 0; }

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
  TileMaps maps;
  if (!get_maps(a.in, a.n_blocks, &maps)) return cudaErrorNotSupported;
  const int grid = 2 * a.n_blocks;
  const size_t sm = sizeof(FusedSmem);
  if (stage == 0) stage_fused_kernel<0><<<grid, FT, sm, st>>>(maps, a);
  else if (stage == 1) stage_fused_kernel<1><<<grid, FT, sm, st>>>(maps, a);
  else stage_fused_kernel<2><<<grid, FT, sm, st>>>(maps, a);
  return cudaGetLastError();
}

}  // namespace batl
