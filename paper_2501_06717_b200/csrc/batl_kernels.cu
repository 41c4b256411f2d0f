// Kernels of the hot path, part 1: plan-driven ghost fill (a1-a4; second-order prolongation, Q-G4b),
// the general stage kernel (a5-a9 for any block: B0 split, body cells, local dt; the reference
// device path), the flux correction at resolution changes (Q-G6b), the dt bookkeeping (a9/a10)
// and the physical-cell scatter/gather used by set/get_state.
// PAPER.md Alg. 2 (L76): gang over blocks, vector over cells -> one CTA per block.
#include "batl_device.cuh"
#include "mhd_physics.cuh"

namespace batl {

__device__ __forceinline__ int sidx(int i, int j, int k) { return ((k + NG) * NS + (j + NG)) * NS + (i + NG); }

// =============================================================== ghost fill ==
// Every ghost cell is written exactly once and only physical cells are read, so a
// single pass with no ordering between messages is enough (Q-G4).
//
// Product kernel: driven by the per-cell plan of batl_grid.hpp.  One CTA per
// destination block; a thread decodes ONE 32-bit plan entry and moves all 8 variables
// of that ghost cell (8 independent loads in flight, then 8 stores), so the index
// arithmetic is paid once per cell, not once per value.  Ghost cells are enumerated
// in storage order: the two k ghost planes are 288 contiguous doubles, j ghost rows
// come in runs of 24, and the x ghosts of adjacent rows pair up into 32-byte runs.
// The plan of a uniform grid is a single 4.9 KB pattern that stays in L1/L2.
// conserved <-> primitive of one cell, IEEE division (the fill of a primitive buffer, general kernel).
// Written with the explicitly rounded intrinsics, which the compiler never contracts into FMAs: equal
// inputs give equal bits at every place these functions are inlined (restrict_prim_cell relies on it).
__device__ __forceinline__ void cell_to_cons(double q[NV], double inv_gm1) {
  const double rho = q[0];
  const double u2 = __dadd_rn(__dadd_rn(__dmul_rn(q[1], q[1]), __dmul_rn(q[2], q[2])), __dmul_rn(q[3], q[3]));
  const double b2 = __dadd_rn(__dadd_rn(__dmul_rn(q[4], q[4]), __dmul_rn(q[5], q[5])), __dmul_rn(q[6], q[6]));
  q[7] = __dadd_rn(__dadd_rn(__dmul_rn(q[7], inv_gm1), __dmul_rn(__dmul_rn(0.5, rho), u2)), __dmul_rn(0.5, b2));   // eq. (5)
  q[1] = __dmul_rn(q[1], rho); q[2] = __dmul_rn(q[2], rho); q[3] = __dmul_rn(q[3], rho);
}
__device__ __forceinline__ void cell_to_prim(double q[NV], double gm1) {
  const double rho = q[0];
  const double ux = __ddiv_rn(q[1], rho), uy = __ddiv_rn(q[2], rho), uz = __ddiv_rn(q[3], rho);
  const double u2 = __dadd_rn(__dadd_rn(__dmul_rn(ux, ux), __dmul_rn(uy, uy)), __dmul_rn(uz, uz));
  const double b2 = __dadd_rn(__dadd_rn(__dmul_rn(q[4], q[4]), __dmul_rn(q[5], q[5])), __dmul_rn(q[6], q[6]));
  q[7] = __dmul_rn(gm1, __dadd_rn(__dadd_rn(q[7], -__dmul_rn(__dmul_rn(0.5, rho), u2)), -__dmul_rn(0.5, b2)));
  q[1] = ux; q[2] = uy; q[3] = uz;
}

// Restriction into a buffer that holds PRIMITIVE variables W (buffer B inside a two-stage step).
// Q-G2/Q-G3: the mean is taken of the CONSERVED variables of the 8 children, in the same pairwise
// order.  The ghost value is computed as
//   mean(W) + [ prim(mean(cons(W))) - prim(cons(mean(W))) ]:
// the bracket is the (small) nonlinear part, in which the rounding of the round trips cancels; a
// uniform state gives mean(W) exactly, as the conserved fill does (T1).
__device__ __forceinline__ void restrict_prim_cell(const double* __restrict__ p, double val[NV], double gm1) {
  const double inv_gm1 = 1.0 / gm1;
  double sw[4][NV], su[4][NV];                            // x pairs (y, z) = (0,0) (1,0) (0,1) (1,1): W and U sums
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    const int off = (q & 1) * NS + (q >> 1) * NS * NS;
    double c0[NV], c1[NV];
#pragma unroll
    for (int v = 0; v < NV; ++v) { c0[v] = p[(size_t)v * NCELL + off]; c1[v] = p[(size_t)v * NCELL + off + 1]; }
#pragma unroll
    for (int v = 0; v < NV; ++v) sw[q][v] = c0[v] + c1[v];
    cell_to_cons(c0, inv_gm1);
    cell_to_cons(c1, inv_gm1);
#pragma unroll
    for (int v = 0; v < NV; ++v) su[q][v] = c0[v] + c1[v];
  }
  double um[NV], rt[NV];
#pragma unroll
  for (int v = 0; v < NV; ++v) {
    val[v] = ((sw[0][v] + sw[1][v]) + (sw[2][v] + sw[3][v])) * 0.125;
    um[v] = ((su[0][v] + su[1][v]) + (su[2][v] + su[3][v])) * 0.125;
    rt[v] = val[v];
  }
  cell_to_prim(um, gm1);                                  // prim(mean(cons(W)))
  cell_to_cons(rt, inv_gm1);
  cell_to_prim(rt, gm1);                                  // prim(cons(mean(W)))
#pragma unroll
  for (int v = 0; v < NV; ++v) val[v] += um[v] - rt[v];
}

// NVT variables per thread, starting at v0 (8 from 0: a thread moves the whole cell; 1: one variable)
template <bool PRIM, int NVT>
__device__ __forceinline__ void ghost_cell(const double* const* __restrict__ src_base, double* __restrict__ dstb, uint32_t e,
                                           const int32_t* __restrict__ src_of_slot, const double* __restrict__ bc_cons,
                                           double gm1, int pass, double beta, int v0) {
  const uint32_t sd = e & 2047u, ss = (e >> 11) & 2047u, slot = (e >> 22) & 63u, kind = e >> 28;
  if ((pass == 1 && kind >= PLAN_PROLONG2) || (pass == 2 && kind < PLAN_PROLONG2)) return;
  double* __restrict__ d = dstb + sd;
  double val[NVT];
  if (kind >= PLAN_PROLONG2) {
    // Q-G4b: the coarse cell's MC(beta)-limited linear profile (O-4's limiter, stored conserved
    // variables) at the centre of this fine cell: U_C +- s_d / 4, d = x, y, z in this order
    const double* __restrict__ p = src_base[slot] + (size_t)src_of_slot[slot] * BLOCK_DOUBLES + ss;
    const double qx = (kind & 1u) ? 0.25 : -0.25, qy = (kind & 2u) ? 0.25 : -0.25, qz = (kind & 4u) ? 0.25 : -0.25;
#pragma unroll
    for (int v = 0; v < NVT; ++v) {
      const double* __restrict__ q = p + (size_t)(v0 + v) * NCELL;
      const double c0 = q[0];
      const double sx = mc_limited(c0 - q[-1], q[1] - c0, beta);
      const double sy = mc_limited(c0 - q[-NS], q[NS] - c0, beta);
      const double sz = mc_limited(c0 - q[-NS * NS], q[NS * NS] - c0, beta);
      double x = c0;
      x += qx * sx;
      x += qy * sy;
      x += qz * sz;
      val[v] = x;
    }
  } else if (kind == PLAN_COPY) {
    const double* __restrict__ p = src_base[slot] + (size_t)src_of_slot[slot] * BLOCK_DOUBLES + ss;
#pragma unroll
    for (int v = 0; v < NVT; ++v) val[v] = p[(size_t)(v0 + v) * NCELL];
  } else if (kind == PLAN_RESTRICT) {
    const double* __restrict__ p = src_base[slot] + (size_t)src_of_slot[slot] * BLOCK_DOUBLES + ss;
    if (PRIM && NVT == NV) restrict_prim_cell(p, val, gm1);
    else
#pragma unroll
    for (int v = 0; v < NVT; ++v) {
      // Q-G3: mean of the 8 children, pairs in x, then y, then z
      const double* __restrict__ q = p + (size_t)(v0 + v) * NCELL;
      const double x00 = q[0] + q[1];
      const double x10 = q[NS] + q[NS + 1];
      const double x01 = q[NS * NS] + q[NS * NS + 1];
      const double x11 = q[NS * NS + NS] + q[NS * NS + NS + 1];
      val[v] = ((x00 + x10) + (x01 + x11)) * 0.125;
    }
  } else {
#pragma unroll
    for (int v = 0; v < NVT; ++v) val[v] = bc_cons[(PRIM ? 6 * NV : 0) + ss * NV + v0 + v];   // [6][8] conserved, then [6][8] primitive
  }
#pragma unroll
  for (int v = 0; v < NVT; ++v) d[(size_t)(v0 + v) * NCELL] = val[v];
}

// Ghost cells come in 16-byte aligned x pairs (storage i = 0-1, 2-3, ..., 10-11) and the plan
// lists them in storage order, so a thread takes one PAIR: when both cells are plain copies of
// an aligned source pair (every same-level face, edge and corner) it moves 8 x double2; any
// other pair (restriction, prolongation, boundary states, clamped copies) is done cell by cell.
constexpr int GF_THREADS = NGHOST / 2;     // 608 = 19 warps: one ghost pair per thread, no loop tail
// Position of stored cell (si, sj, sk) among the ghost cells of a block in storage order (the order of
// the plan entries); the cell must be a ghost cell.
__device__ __forceinline__ int ghost_ordinal(int si, int sj, int sk) {
  if (sk < NG) return sk * NS * NS + sj * NS + si;
  if (sk >= NG + NI) return 2 * NS * NS + NI * 80 + (sk - NG - NI) * NS * NS + sj * NS + si;
  const int base = 2 * NS * NS + (sk - NG) * 80;          // 80 ghost cells in a plane with physical cells
  if (sj < NG) return base + sj * NS + si;
  if (sj >= NG + NI) return base + 2 * NS + NI * 4 + (sj - NG - NI) * NS + si;
  return base + 2 * NS + (sj - NG) * 4 + (si < NG ? si : si - NI);
}

// FACES: the pass after a stage on the product path.  The same-level faces have been written by the
// neighbours' stage kernels and the scheme reads no edge or corner ghost, so only the face ghosts at
// resolution changes and boundaries are left: one CTA of 64 threads per (block, face), which leaves at
// once if a same-level neighbour writes that face; thread t takes the t-th x pair of the face slab.
// In the FACES pass over a conserved buffer a thread moves ONE variable of its pair (512 threads per face):
// the few faces at resolution changes are latency-bound (a restricted ghost cell reads 8 fine cells), and
// eight times the threads hide it.
template <bool PRIM, bool FACES>
__global__ void __launch_bounds__(FACES ? (PRIM ? 64 : 64 * NV) : GF_THREADS) ghost_fill_kernel(double* __restrict__ S, const uint32_t* __restrict__ plan,
                                                         const int32_t* __restrict__ plan_id,
                                                         const int32_t* __restrict__ plan_src,
                                                         const double* __restrict__ bc_cons,
                                                         const int32_t* __restrict__ list, double gm1,
                                                         const int32_t* __restrict__ push_nbr, int pass, double beta,
                                                         const int32_t* __restrict__ owner, double* const* __restrict__ peer) {
  __shared__ int32_t src_of_slot[PLAN_SLOTS];
  __shared__ const double* src_base[PLAN_SLOTS];           // buffer that holds the source block of a slot (sharded: its owner's)
  // Blocks are walked from the last to the first: the stage kernel before this fill walks them
  // upwards, so the blocks it wrote last are still in the 126 MB L2 when the fill starts, and the
  // fill leaves the low-numbered blocks there for the stage kernel that follows.
  const int q = gridDim.x - 1 - blockIdx.x;
  const int b = list ? list[q] : q;
  constexpr int NVT = (FACES && !PRIM) ? 1 : NV;           // variables per thread
  const int v0 = (FACES && !PRIM) ? threadIdx.x >> 6 : 0;
  int pair_index = threadIdx.x;
  if (FACES) {
    const int f = blockIdx.y, t = threadIdx.x & 63;
    const int32_t pn = push_nbr[(size_t)b * 6 + f];
    if (pn >= 0 || pn == PUSH_BY_COARSER) return;           // a neighbour's stage kernel writes this face
    int si, sj, sk;                                          // first cell of the pair, storage coordinates
    if (f < 2) { si = f ? NG + NI : 0; sj = NG + (t & 7); sk = NG + (t >> 3); }
    else if (f < 4) { si = NG + 2 * (t & 3); sj = (f & 1 ? NG + NI : 0) + ((t >> 2) & 1); sk = NG + (t >> 3); }
    else { si = NG + 2 * (t & 3); sj = NG + ((t >> 2) & 7); sk = (f & 1 ? NG + NI : 0) + (t >> 5); }
    pair_index = ghost_ordinal(si, sj, sk) >> 1;
  }
  if (threadIdx.x < PLAN_SLOTS) {
    const int32_t sb = plan_src[(size_t)b * PLAN_SLOTS + threadIdx.x];
    src_of_slot[threadIdx.x] = sb;
    src_base[threadIdx.x] = (owner && sb >= 0) ? peer[owner[sb]] : S;
  }
  const uint2* __restrict__ P = reinterpret_cast<const uint2*>(plan + (size_t)plan_id[b] * NGHOST);
  double* __restrict__ dstb = S + (size_t)b * BLOCK_DOUBLES;
  __syncthreads();
  {
    const uint2 e = P[pair_index];
    // same kind (copy) and slot, source and destination cells consecutive, both pairs aligned
    const bool pair = ((e.x ^ e.y) >> 22) == 0 && (e.x >> 28) == PLAN_COPY &&
                      (e.y & 0x3FFFFFu) == (e.x & 0x3FFFFFu) + 0x801u && (e.x & 0x801u) == 0;
    if (pair && pass != 2) {
      const uint32_t sd = e.x & 2047u, ss = (e.x >> 11) & 2047u, slot = (e.x >> 22) & 63u;
      const double2* __restrict__ p = reinterpret_cast<const double2*>(src_base[slot] + (size_t)src_of_slot[slot] * BLOCK_DOUBLES + ss);
      double2* __restrict__ d = reinterpret_cast<double2*>(dstb + sd);
      double2 val[NVT];
#pragma unroll
      for (int v = 0; v < NVT; ++v) val[v] = p[(size_t)(v0 + v) * (NCELL / 2)];
#pragma unroll
      for (int v = 0; v < NVT; ++v) d[(size_t)(v0 + v) * (NCELL / 2)] = val[v];
    } else if (!pair) {
      ghost_cell<PRIM, NVT>(src_base, dstb, e.x, src_of_slot, bc_cons, gm1, pass, beta, v0);
      ghost_cell<PRIM, NVT>(src_base, dstb, e.y, src_of_slot, bc_cons, gm1, pass, beta, v0);
    }
  }
}

cudaError_t launch_ghost_fill(double* state, const uint32_t* plan, const int32_t* plan_id, const int32_t* plan_src,
                              const double* bc_cons, const int32_t* list, int n_blocks, cudaStream_t st,
                              bool prim, double gamma, const int32_t* push_nbr, int pass, double beta,
                              const int32_t* owner, double* const* peer_state) {
  if (n_blocks == 0) return cudaSuccess;
  if (push_nbr) {                                          // faces that no same-level neighbour writes
    const dim3 grid(n_blocks, 6);
    if (prim) ghost_fill_kernel<true, true><<<grid, 64, 0, st>>>(state, plan, plan_id, plan_src, bc_cons, list, gamma - 1.0, push_nbr, pass, beta, owner, peer_state);
    else ghost_fill_kernel<false, true><<<grid, 64 * NV, 0, st>>>(state, plan, plan_id, plan_src, bc_cons, list, 0.0, push_nbr, pass, beta, owner, peer_state);
  } else if (prim) {
    ghost_fill_kernel<true, false><<<n_blocks, GF_THREADS, 0, st>>>(state, plan, plan_id, plan_src, bc_cons, list, gamma - 1.0, push_nbr, pass, beta, owner, peer_state);
  } else {
    ghost_fill_kernel<false, false><<<n_blocks, GF_THREADS, 0, st>>>(state, plan, plan_id, plan_src, bc_cons, list, 0.0, push_nbr, pass, beta, owner, peer_state);
  }
  return cudaGetLastError();
}

// Reference kernel (kernel variant 1): walks the message records directly, one value
// per thread-iteration.  Slow (index decoding per value); kept as the device-side
// cross-check of the plan expansion.
__global__ void __launch_bounds__(256) ghost_fill_msg_kernel(double* __restrict__ S, const batl_ghost_msg* __restrict__ msg,
                                                             const int32_t* __restrict__ msg_start,
                                                             const double* __restrict__ bc_cons) {
  const int b = blockIdx.x;
  const int m0 = msg_start[b], m1 = msg_start[b + 1];
  double* __restrict__ dstb = S + (size_t)b * BLOCK_DOUBLES;
  for (int mi = m0; mi < m1; ++mi) {
    const batl_ghost_msg m = msg[mi];
    const int n0 = m.n[0], n1 = m.n[1], n2 = m.n[2];
    const int cells = n0 * n1 * n2;
    const int items = cells * NV;
    const double* __restrict__ srcb = (m.src >= 0) ? S + (size_t)m.src * BLOCK_DOUBLES : nullptr;
    for (int it = threadIdx.x; it < items; it += blockDim.x) {
      int r = it;
      const int ii = r % n0; r /= n0;
      const int jj = r % n1; r /= n1;
      const int kk = r % n2;
      const int v = r / n2;
      const int ci = m.lo[0] + ii, cj = m.lo[1] + jj, ck = m.lo[2] + kk;
      double val;
      if (m.kind == BATL_MSG_FIXED) {
        val = bc_cons[(-2 - m.src) * NV + v];
      } else {
        const int si = (m.mul[0] * ci + m.off[0]) >> m.shift[0];
        const int sj = (m.mul[1] * cj + m.off[1]) >> m.shift[1];
        const int sk = (m.mul[2] * ck + m.off[2]) >> m.shift[2];
        const double* __restrict__ p = srcb + (size_t)v * NCELL + sidx(si, sj, sk);
        if (m.kind == BATL_MSG_RESTRICT) {
          const double x00 = p[0] + p[1];
          const double x10 = p[NS] + p[NS + 1];
          const double x01 = p[NS * NS] + p[NS * NS + 1];
          const double x11 = p[NS * NS + NS] + p[NS * NS + NS + 1];
          val = ((x00 + x10) + (x01 + x11)) * 0.125;
        } else {
          val = p[0];
        }
      }
      dstb[(size_t)v * NCELL + sidx(ci, cj, ck)] = val;
    }
  }
}

cudaError_t launch_ghost_fill_msg(double* state, const batl_ghost_msg* msg, const int32_t* msg_start,
                                  const double* bc_cons, int n_blocks, cudaStream_t st) {
  if (n_blocks == 0) return cudaSuccess;
  ghost_fill_msg_kernel<<<n_blocks, 256, 0, st>>>(state, msg, msg_start, bc_cons);
  return cudaGetLastError();
}

// ==================================================== physical-cell scatter/gather ==
__global__ void __launch_bounds__(512) scatter_phys_kernel(const double* __restrict__ compact, double* __restrict__ S) {
  const int b = blockIdx.x, t = threadIdx.x;
  const int i = t & 7, j = (t >> 3) & 7, k = t >> 6;
#pragma unroll
  for (int v = 0; v < NV; ++v)
    S[((size_t)b * NV + v) * NCELL + sidx(i, j, k)] = compact[((size_t)b * NV + v) * NPHYS + t];
}
__global__ void __launch_bounds__(512) gather_phys_kernel(const double* __restrict__ S, double* __restrict__ compact) {
  const int b = blockIdx.x, t = threadIdx.x;
  const int i = t & 7, j = (t >> 3) & 7, k = t >> 6;
#pragma unroll
  for (int v = 0; v < NV; ++v)
    compact[((size_t)b * NV + v) * NPHYS + t] = S[((size_t)b * NV + v) * NCELL + sidx(i, j, k)];
}
cudaError_t launch_scatter_phys(const double* compact, double* state, int n_blocks, cudaStream_t st) {
  if (n_blocks == 0) return cudaSuccess;
  scatter_phys_kernel<<<n_blocks, 512, 0, st>>>(compact, state);
  return cudaGetLastError();
}
cudaError_t launch_gather_phys(const double* state, double* compact, int n_blocks, cudaStream_t st) {
  if (n_blocks == 0) return cudaSuccess;
  gather_phys_kernel<<<n_blocks, 512, 0, st>>>(state, compact);
  return cudaGetLastError();
}

// ================================================================ dt bookkeeping ==
// Q-T2 (lagged global dt): the dt of step n is the minimum of dt_c over the faces
// evaluated in stage 2 of step n-1 (stage 0 for n = 0).  One thread; keeps the
// whole multi-step loop on the device.
__global__ void tick_kernel(DevScalars* sc, int mode, int dt_mode, double dt_fixed) {
  if (mode == 1) {                                  // end of a step
    sc->dt_last = sc->dt;
    if (dt_mode != BATL_DT_LOCAL) sc->t += sc->dt;
  }
  if (dt_mode == BATL_DT_GLOBAL) {
    sc->dt = __longlong_as_double((long long)sc->dt_next_bits);
    sc->dt_next_bits = 0x7FF0000000000000ull;       // +inf
  } else if (dt_mode == BATL_DT_FIXED) {
    sc->dt = dt_fixed;
  } else {
    sc->dt = 0.0;
  }
}
__global__ void reset_scalars_kernel(DevScalars* sc) {
  sc->dt = 0.0; sc->dt_last = 0.0; sc->t = 0.0;
  sc->dt_next_bits = 0x7FF0000000000000ull;
  sc->warn = 0; sc->pad = 0;
}
cudaError_t launch_tick(DevScalars* sc, int mode, int dt_mode, double dt_fixed, cudaStream_t st) {
  tick_kernel<<<1, 1, 0, st>>>(sc, mode, dt_mode, dt_fixed);
  return cudaGetLastError();
}
cudaError_t launch_reset_scalars(DevScalars* sc, cudaStream_t st) {
  reset_scalars_kernel<<<1, 1, 0, st>>>(sc);
  return cudaGetLastError();
}

// ========================================================== general stage kernel ==
// One CTA per block, one thread per physical cell.  The 12^3 x 8 tile is converted to
// primitives in shared memory; every thread then evaluates the six faces of its cell
// (each face is therefore computed twice per block).  Handles every option (B0 split,
// body, local dt); it is the reference device path and serves the blocks the fused
// kernel (batl_stage_fused.cu) does not cover.
constexpr int GEN_THREADS = 512;
constexpr size_t GEN_SMEM = BLOCK_BYTES + NCELL;   // W[8][1728] + body[1728]

struct FaceResult { double F[NV]; double Bn; double c; };

template <int D>
__device__ __forceinline__ void general_face(const double* __restrict__ W, const unsigned char* __restrict__ body,
                                             int sL, const double B0f[3], const StageArgs& a, double inv_gm1,
                                             FaceResult& o) {
  constexpr int st = (D == 0) ? 1 : (D == 1) ? NS : NS * NS;
  const int sR = sL + st;
  const bool bL = body[sL], bR = body[sR];
#pragma unroll
  for (int v = 0; v < NV; ++v) o.F[v] = 0.0;
  o.Bn = 0.0; o.c = 0.0;
  if (bL && bR) return;                                   // Q-F3: faces inside the body are skipped
  const bool nearL = body[sL - st] || bL || bR;           // Q-R3: zero slope next to the body
  const bool nearR = bL || bR || body[sR + st];
  double WL[NV], WR[NV];
#pragma unroll
  for (int v = 0; v < NV; ++v) {
    const double* __restrict__ w = W + v * NCELL;
    const double wm = w[sL - st], wl = w[sL], wr = w[sR], wp = w[sR + st];
    const double dc = wr - wl;
    const double slL = nearL ? 0.0 : mc_limited(wl - wm, dc, a.beta);
    const double slR = nearR ? 0.0 : mc_limited(dc, wp - wr, a.beta);
    WL[v] = wl + 0.5 * slL;                               // W^L_{c+1/2}
    WR[v] = wr - 0.5 * slR;                               // W^R_{c+1/2}
  }
  if (bL || bR) {                                         // Q-F3: fixed-density reflective body state
    double* Wb = bL ? WL : WR;
    const double* Wt = bL ? WR : WL;
    Wb[0] = a.rho_body;
    Wb[1] = -Wt[1]; Wb[2] = -Wt[2]; Wb[3] = -Wt[3];
    Wb[4] = Wt[4]; Wb[5] = Wt[5]; Wb[6] = Wt[6];
    Wb[7] = (a.p_body > 0.0) ? a.p_body : Wt[7];
  }
  rusanov_flux<D>(WL, WR, B0f, a.gamma, inv_gm1, o.F, o.Bn, o.c, a.flux_type);
}

// Q-G6b: keep the flux through face cell (t_lo, t_hi) of face f of block b if that face is at a resolution change
__device__ __forceinline__ void save_face_flux(const StageArgs& a, int b, int f, int t_lo, int t_hi, const double F[NV]) {
  const int slot = a.fc_slot[(size_t)b * 6 + f];
  if (slot < 0) return;
  double* __restrict__ o = a.fc_buf + (size_t)slot * NV * NI * NI + t_hi * NI + t_lo;
#pragma unroll
  for (int v = 0; v < NV; ++v) o[v * NI * NI] = F[v];
}

__device__ __forceinline__ void b0_at(const StageArgs& a, double x, double y, double z, double B0[3]) {
  if (a.use_b0 == 2) { B0[0] = a.m[0]; B0[1] = a.m[1]; B0[2] = a.m[2]; }
  else dipole_field(a.m, x, y, z, B0);
}

template <int STAGE>
__global__ void __launch_bounds__(GEN_THREADS, 1) stage_general_kernel(const StageArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double* W = reinterpret_cast<double*>(smem_raw);                  // [8][1728] primitives
  unsigned char* body = smem_raw + BLOCK_BYTES;                     // [1728]
  __shared__ double red[GEN_THREADS / 32];

  const int b = a.blocks ? a.blocks[blockIdx.x] : blockIdx.x, tid = threadIdx.x;
  const BlockGeom G = a.geom[b];
  const double* __restrict__ Uin = a.in + (size_t)b * BLOCK_DOUBLES;
  const bool has_body = a.use_body && (G.flags & 1);
  const uint32_t* __restrict__ mask = has_body ? a.body_mask + (size_t)G.mask_slot * BODY_MASK_WORDS : nullptr;
  const double gm1 = a.gamma - 1.0, inv_gm1 = 1.0 / gm1;
  int warn = 0;

  // ---- O-3: primitives of every stored cell
  for (int s = tid; s < NCELL; s += GEN_THREADS) {
    const bool isb = has_body && ((mask[s >> 5] >> (s & 31)) & 1u);
    body[s] = isb;
    const bool prim_in = STAGE == 2 && a.b_prim;            // buffer B: stage 1 stored primitives
    const double rho = Uin[s];
    double ux = Uin[1 * NCELL + s], uy = Uin[2 * NCELL + s], uz = Uin[3 * NCELL + s];
    if (!prim_in) { ux /= rho; uy /= rho; uz /= rho; }
    const double bx = Uin[4 * NCELL + s], by = Uin[5 * NCELL + s], bz = Uin[6 * NCELL + s];
    const double u2 = ux * ux + uy * uy + uz * uz;
    const double b2 = bx * bx + by * by + bz * bz;
    const double p = prim_in ? Uin[7 * NCELL + s] : gm1 * (Uin[7 * NCELL + s] - 0.5 * rho * u2 - 0.5 * b2);
    W[s] = rho; W[NCELL + s] = ux; W[2 * NCELL + s] = uy; W[3 * NCELL + s] = uz;
    W[4 * NCELL + s] = bx; W[5 * NCELL + s] = by; W[6 * NCELL + s] = bz; W[7 * NCELL + s] = p;
    const int si = s % NS, sj = (s / NS) % NS, sk = s / (NS * NS);
    const bool phys = si >= NG && si < NG + NI && sj >= NG && sj < NG + NI && sk >= NG && sk < NG + NI;
    if (phys && !isb) {
      if (!isfinite(rho) || !isfinite(p)) warn |= BATL_WARN_NONFINITE;
      if (rho <= 0.0 || p <= 0.0) warn |= BATL_WARN_NEGATIVE;
    }
  }
  __syncthreads();

  const int i = tid & 7, j = (tid >> 3) & 7, k = tid >> 6;
  const int sc = sidx(i, j, k);
  const bool cell_is_body = body[sc];
  double dt_c = __longlong_as_double(0x7FF0000000000000ll);
  if (!cell_is_body) {
    double R[NV];
#pragma unroll
    for (int v = 0; v < NV; ++v) R[v] = 0.0;
    double divB1 = 0.0, speed = 0.0;
    double dB0[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};   // dB0[comp][dir]
    const double xc = G.x0[0] + (i + 0.5) * G.D[0], yc = G.x0[1] + (j + 0.5) * G.D[1], zc = G.x0[2] + (k + 0.5) * G.D[2];
    FaceResult fm, fp;
    double B0m[3] = {0, 0, 0}, B0p[3] = {0, 0, 0};
    // x faces
    if (a.use_b0) { b0_at(a, G.x0[0] + i * G.D[0], yc, zc, B0m); b0_at(a, G.x0[0] + (i + 1) * G.D[0], yc, zc, B0p); }
    general_face<0>(W, body, sc - 1, B0m, a, inv_gm1, fm);
    general_face<0>(W, body, sc, B0p, a, inv_gm1, fp);
    if (a.fc_slot && i == 0) save_face_flux(a, b, 0, j, k, fm.F);
    if (a.fc_slot && i == NI - 1) save_face_flux(a, b, 1, j, k, fp.F);
#pragma unroll
    for (int v = 0; v < NV; ++v) R[v] -= (fp.F[v] - fm.F[v]) * G.invD[0];
    divB1 += (fp.Bn - fm.Bn) * G.invD[0];
    speed += fmax(fm.c, fp.c) * G.invD[0];
#pragma unroll
    for (int c = 0; c < 3; ++c) dB0[c][0] = (B0p[c] - B0m[c]) * G.invD[0];
    // y faces
    if (a.use_b0) { b0_at(a, xc, G.x0[1] + j * G.D[1], zc, B0m); b0_at(a, xc, G.x0[1] + (j + 1) * G.D[1], zc, B0p); }
    general_face<1>(W, body, sc - NS, B0m, a, inv_gm1, fm);
    general_face<1>(W, body, sc, B0p, a, inv_gm1, fp);
    if (a.fc_slot && j == 0) save_face_flux(a, b, 2, i, k, fm.F);
    if (a.fc_slot && j == NI - 1) save_face_flux(a, b, 3, i, k, fp.F);
#pragma unroll
    for (int v = 0; v < NV; ++v) R[v] -= (fp.F[v] - fm.F[v]) * G.invD[1];
    divB1 += (fp.Bn - fm.Bn) * G.invD[1];
    speed += fmax(fm.c, fp.c) * G.invD[1];
#pragma unroll
    for (int c = 0; c < 3; ++c) dB0[c][1] = (B0p[c] - B0m[c]) * G.invD[1];
    // z faces
    if (a.use_b0) { b0_at(a, xc, yc, G.x0[2] + k * G.D[2], B0m); b0_at(a, xc, yc, G.x0[2] + (k + 1) * G.D[2], B0p); }
    general_face<2>(W, body, sc - NS * NS, B0m, a, inv_gm1, fm);
    general_face<2>(W, body, sc, B0p, a, inv_gm1, fp);
    if (a.fc_slot && k == 0) save_face_flux(a, b, 4, i, j, fm.F);
    if (a.fc_slot && k == NI - 1) save_face_flux(a, b, 5, i, j, fp.F);
#pragma unroll
    for (int v = 0; v < NV; ++v) R[v] -= (fp.F[v] - fm.F[v]) * G.invD[2];
    divB1 += (fp.Bn - fm.Bn) * G.invD[2];
    speed += fmax(fm.c, fp.c) * G.invD[2];
#pragma unroll
    for (int c = 0; c < 3; ++c) dB0[c][2] = (B0p[c] - B0m[c]) * G.invD[2];

    // ---- O-6: sources from the cell-centre state of the stage input
    const double ux = W[NCELL + sc], uy = W[2 * NCELL + sc], uz = W[3 * NCELL + sc];
    const double bx = W[4 * NCELL + sc], by = W[5 * NCELL + sc], bz = W[6 * NCELL + sc];
    double B0c[3] = {0, 0, 0};
    if (a.use_b0) b0_at(a, xc, yc, zc, B0c);
    if (a.use_divb) {                                       // 8-wave terms, RHS of eqs (2)-(4)
      R[1] -= (bx + B0c[0]) * divB1; R[2] -= (by + B0c[1]) * divB1; R[3] -= (bz + B0c[2]) * divB1;
      R[4] -= ux * divB1; R[5] -= uy * divB1; R[6] -= uz * divB1;
      R[7] -= (ux * bx + uy * by + uz * bz) * divB1;
    }
    if (a.use_b0) {                                         // Q-S2
      const double divB0 = dB0[0][0] + dB0[1][1] + dB0[2][2];
      const double cx = dB0[2][1] - dB0[1][2], cy = dB0[0][2] - dB0[2][0], cz = dB0[1][0] - dB0[0][1];
      const double sx = -bx * divB0 - (cy * bz - cz * by);
      const double sy = -by * divB0 - (cz * bx - cx * bz);
      const double sz = -bz * divB0 - (cx * by - cy * bx);
      R[1] += sx; R[2] += sy; R[3] += sz;
      R[7] += ux * sx + uy * sy + uz * sz;
    }
    dt_c = a.cfl / speed;                                   // O-8
    if (STAGE != 0) {
      double dt;
      if (a.dt_mode == BATL_DT_LOCAL) {                     // Q-T3
        double* dtl = a.dt_local + (size_t)b * NPHYS + tid;
        if (STAGE == 1 || STAGE == 3) *dtl = dt_c;
        dt = (STAGE == 1 || STAGE == 3) ? dt_c : *dtl;
      } else {
        dt = a.sc->dt;
      }
      const double f = (STAGE == 1 ? 0.5 : 1.0) * dt;
      double Un[NV];
#pragma unroll
      for (int v = 0; v < NV; ++v) Un[v] = a.base[((size_t)b * NV + v) * NCELL + sc] + f * R[v];   // O-7
      if (STAGE == 1 && a.b_prim) cell_to_prim(Un, gm1);
      double* __restrict__ o = a.out + (size_t)b * BLOCK_DOUBLES + sc;
#pragma unroll
      for (int v = 0; v < NV; ++v) o[(size_t)v * NCELL] = Un[v];
      if (a.push_nbr) { int pn[3]; push_targets(a.push_nbr + (size_t)b * 6, i, j, k, pn); push_cell(a, o, pn, b, i, j, k, Un); }
    }
  } else if (STAGE != 0) {
    if (a.fc_slot) {                                        // a body cell takes no flux: keep the buffer defined
      const double Z[NV] = {0, 0, 0, 0, 0, 0, 0, 0};
      if (i == 0) save_face_flux(a, b, 0, j, k, Z);
      if (i == NI - 1) save_face_flux(a, b, 1, j, k, Z);
      if (j == 0) save_face_flux(a, b, 2, i, k, Z);
      if (j == NI - 1) save_face_flux(a, b, 3, i, k, Z);
      if (k == 0) save_face_flux(a, b, 4, i, j, Z);
      if (k == NI - 1) save_face_flux(a, b, 5, i, j, Z);
    }
    double Un[NV];
#pragma unroll
    for (int v = 0; v < NV; ++v) Un[v] = a.base[((size_t)b * NV + v) * NCELL + sc];
    if (STAGE == 1 && a.b_prim) cell_to_prim(Un, gm1);
    double* __restrict__ o = a.out + (size_t)b * BLOCK_DOUBLES + sc;
#pragma unroll
    for (int v = 0; v < NV; ++v) o[(size_t)v * NCELL] = Un[v];
    if (a.push_nbr) { int pn[3]; push_targets(a.push_nbr + (size_t)b * 6, i, j, k, pn); push_cell(a, o, pn, b, i, j, k, Un); }
  }

  // ---- a9: block minimum of dt_c, one atomic per block
  if (STAGE != 1 && a.dt_mode == BATL_DT_GLOBAL) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) dt_c = fmin(dt_c, __shfl_xor_sync(0xffffffffu, dt_c, o));
    if ((tid & 31) == 0) red[tid >> 5] = dt_c;
    __syncthreads();
    if (tid < 32) {
      double v = (tid < GEN_THREADS / 32) ? red[tid] : __longlong_as_double(0x7FF0000000000000ll);
#pragma unroll
      for (int o = 8; o > 0; o >>= 1) v = fmin(v, __shfl_xor_sync(0xffffffffu, v, o));
      if (tid == 0) atomic_min_positive(&a.sc->dt_next_bits, v);
    }
  }
  if (warn) atomicOr(&a.sc->warn, warn);
}

cudaError_t launch_stage_general(int stage, const StageArgs& a, cudaStream_t st) {
  const int n = a.blocks ? a.n_list : a.n_blocks;         // one CTA per block of the list (or per block)
  if (n == 0) return cudaSuccess;
  if (stage == 0) stage_general_kernel<0><<<n, GEN_THREADS, GEN_SMEM, st>>>(a);
  else if (stage == 1) stage_general_kernel<1><<<n, GEN_THREADS, GEN_SMEM, st>>>(a);
  else if (stage == 2) stage_general_kernel<2><<<n, GEN_THREADS, GEN_SMEM, st>>>(a);
  else stage_general_kernel<3><<<n, GEN_THREADS, GEN_SMEM, st>>>(a);
  return cudaGetLastError();
}

// ============================================================= flux correction ==
// Q-G6b ("nearly conservative form"): after a stage, the cells of a
// block next to a face that borders FINER blocks exchange the flux they used through that face for the
// mean of the four fine fluxes that cover it, U += -+ f dt / D (mean - own).  One CTA per block with
// such faces, one thread per (variable, face cell); the corrected cell is written again into the face
// ghosts of the same-level neighbours that see it.
__global__ void __launch_bounds__(NV * NI * NI) flux_correct_kernel(const StageArgs a, const int stage,
                                                                    const int32_t* __restrict__ fc_list,
                                                                    const int32_t* __restrict__ fc_group) {
  const int r0 = fc_group[2 * blockIdx.x], nr = fc_group[2 * blockIdx.x + 1];
  const int v = threadIdx.x >> 6, t = threadIdx.x & 63, t_lo = t & 7, t_hi = t >> 3;
  // the faces of one block one after the other: a cell at an edge or corner of the block is corrected
  // through two or three of them, always in the same order
  for (int r = r0; r < r0 + nr; ++r) {
    const int32_t* __restrict__ rec = fc_list + (size_t)r * 8;
    const int b = rec[0], f = rec[1], own = rec[2];
    const int d = f >> 1, side = f & 1;
    int c[3];
    c[d] = side ? NI - 1 : 0;
    c[d == 0 ? 1 : 0] = t_lo;
    c[d == 2 ? 1 : 2] = t_hi;
    const BlockGeom& G = a.geom[b];
    const int sc = sidx(c[0], c[1], c[2]);
    bool body = false;                                      // body cells are never updated (Q-F3)
    if (a.use_body && (G.flags & 1)) {
      const uint32_t* __restrict__ mask = a.body_mask + (size_t)G.mask_slot * BODY_MASK_WORDS;
      body = (mask[sc >> 5] >> (sc & 31)) & 1u;
    }
    if (!body) {
      const double Fo = a.fc_buf[((size_t)own * NV + v) * (NI * NI) + t];
      const int fs = rec[3 + (t_lo >> 2) + 2 * (t_hi >> 2)];
      const double* __restrict__ F4 = a.fc_buf + ((size_t)fs * NV + v) * (NI * NI) + 2 * (t_hi & 3) * NI + 2 * (t_lo & 3);
      const double m = ((F4[0] + F4[1]) + (F4[NI] + F4[NI + 1])) * 0.25;   // pairs along the lower tangential axis first
      const double dt = (a.dt_mode == BATL_DT_LOCAL) ? a.dt_local[(size_t)b * NPHYS + (c[2] * NI + c[1]) * NI + c[0]] : a.sc->dt;
      const double fac = (stage == 1 ? 0.5 : 1.0) * dt;
      double* __restrict__ o = a.out + (size_t)b * BLOCK_DOUBLES + (size_t)v * NCELL + sc;
      const double val = *o + (side ? -1.0 : 1.0) * fac * G.invD[d] * (m - Fo);
      *o = val;
      if (a.push_nbr) {
        int pn[3];
        push_targets(a.push_nbr + (size_t)b * 6, c[0], c[1], c[2], pn);
        const ptrdiff_t sh[3] = {c[0] < NG ? NI : -NI, c[1] < NG ? NI * NS : -NI * NS, c[2] < NG ? NI * NS * NS : -NI * NS * NS};
#pragma unroll
        for (int q = 0; q < 3; ++q)
          if (pn[q] >= 0) o[(ptrdiff_t)(pn[q] - b) * (ptrdiff_t)BLOCK_DOUBLES + sh[q]] = val;
      }
    }
    __syncthreads();
  }
}

cudaError_t launch_flux_correction(int stage, const StageArgs& a, const int32_t* fc_list, const int32_t* fc_group,
                                   int n_groups, cudaStream_t st) {
  if (n_groups == 0) return cudaSuccess;
  flux_correct_kernel<<<n_groups, NV * NI * NI, 0, st>>>(a, stage, fc_list, fc_group);
  return cudaGetLastError();
}

cudaError_t init_kernel_attributes() {
  cudaError_t e;
  e = cudaFuncSetAttribute(stage_general_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)GEN_SMEM);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(stage_general_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)GEN_SMEM);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(stage_general_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)GEN_SMEM);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(stage_general_kernel<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)GEN_SMEM);
  if (e != cudaSuccess) return e;
  return cudaSuccess;   // the fused kernels set theirs per instantiation at the first launch
}

}  // namespace batl
