// Device-side data structures and kernel launchers shared by batl_api.cu and the
// kernel translation units.  sm_100a only.
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

#include "batl_grid.hpp"

namespace batl {

// scalars that live in device memory so that a whole mhd_step(n) needs no host sync
struct DevScalars {
  double dt;                         // time step of the step being computed
  double dt_last;                    // time step of the last completed step
  double t;                          // simulation time
  unsigned long long dt_next_bits;   // running minimum of dt_c (bit pattern of a positive double)
  int warn;                          // BATL_WARN_* bits
  int pad;
};

// everything a stage kernel needs; passed by value
struct StageArgs {
  const double* in;                  // state the fluxes are computed from (12^3 tiles)
  const double* base;                // U^n (only physical cells are read)
  double* out;                       // receives the physical cells of the stage result
  const BlockGeom* geom;
  const uint32_t* body_mask;
  double* dt_local;                  // [nB][512] (dt_mode local) or nullptr
  DevScalars* sc;
  double gamma, cfl, beta;
  double gm1, inv_gm1, half_beta;    // gamma - 1, 1 / (gamma - 1), beta / 2 (host-computed: no registers spent on them)
  double m[3];                       // dipole moment (use_b0 = 1) or uniform B0 (use_b0 = 2)
  double rho_body, p_body;
  int dt_mode, use_divb, use_b0, use_body;
  int n_order;                       // 1: piecewise-constant face states (Q-U2)
  int flux_type;                     // 0 Rusanov, 1 HLL-type (Q-F4)
  int b_prim;                        // 1: the intermediate state U* (buffer B) is stored as PRIMITIVE variables:
                                     // stage 1 writes (rho, u, B1, p), stage 2 reads them (the fused kernels
                                     // always do; the general kernel follows this flag)
  int n_blocks;
  int n_sm;                          // SM count of the device the grid is bound on
  const int32_t* blocks;             // blocks this launch processes (device), nullptr = all n_blocks
  int n_list;                        // length of `blocks`
  const int32_t* push_nbr;           // [nB][6] same-level face neighbours whose ghost slots this launch writes
                                     // (batl_grid.hpp), nullptr = no pushing (reference path)
  const int32_t* push_fine;          // [n][4] finer neighbours of the faces with push_nbr = -2 - n
  // flux correction (Q-G6b): slots of the faces at resolution changes (batl_grid.hpp), nullptr = off; the
  // stage kernels store the flux through every face cell of such a face in fc_buf[slot][var][t_hi][t_lo]
  const int32_t* fc_slot;            // [nB][6]
  double* fc_buf;
  int fused_body;                    // 1: this launch of the fused kernel takes the blocks with body cells too
  // sharding (batl.h, batl_set_partition): owner[b] = rank that owns block b, nullptr = one GPU; peer_out[r] /
  // peer_in[r] = the buffers `out` / `in` of rank r as mapped into this process
  const int32_t* owner;
  double* const* peer_out;
  int rank;
};

// Ghost cells without a fill pass (the ghost layer "must be filled
// in every time"): the thread that has just computed physical cell (i, j, k) of block b also writes
// it into the face-ghost slot of the same-level neighbour that sees it as a ghost cell.
// o = address of variable 0 of the cell in the output buffer, nb = the block's row of push_nbr.
// push_targets reads the (up to three) neighbour ids first, so that their latency does not sit
// between the stores; n[d] < 0: nothing to write in direction d.
__device__ __forceinline__ void push_targets(const int32_t* nb, int i, int j, int k, int n[3]) {
  n[0] = (i < NG || i >= NI - NG) ? nb[i < NG ? 0 : 1] : -1;
  n[1] = (j < NG || j >= NI - NG) ? nb[j < NG ? 2 : 3] : -1;
  n[2] = (k < NG || k >= NI - NG) ? nb[k < NG ? 4 : 5] : -1;
}
// o = address of variable 0 of the cell in the output buffer `out` of this rank.  Sharded (a.owner): a
// neighbour block that lives on another GPU is written through that rank's mapped buffer (same block and
// cell offsets: every rank's buffer has room for the whole grid).
__device__ __forceinline__ double* push_base(const StageArgs& a, int nb) {
  if (a.owner) {
    const int rk = a.owner[nb];
    if (rk != a.rank) return a.peer_out[rk];
  }
  return a.out;
}
// FINE: the grid may have faces with finer neighbours whose ghosts are pushed (a.push_fine != nullptr; the
// fused kernel's AMR variants); without it the code is the same-level copy alone, and the uniform-grid path
// pays nothing for the other
template <bool FINE>
__device__ __forceinline__ void push_cell_t(const StageArgs& a, double* __restrict__ o, const int n[3], int b, int i, int j, int k,
                                            const double U[NV]) {
  const int c[3] = {i, j, k};
  const ptrdiff_t st[3] = {1, NS, NS * NS};
#pragma unroll
  for (int q = 0; q < 3; ++q) {
    if (n[q] >= 0) {                                       // same level: the cell is a face ghost of that neighbour
      double* __restrict__ d = push_base(a, n[q]) + (o - a.out) + (ptrdiff_t)(n[q] - b) * (ptrdiff_t)BLOCK_DOUBLES +
                               (c[q] < NG ? NI : -NI) * st[q];
#pragma unroll
      for (int v = 0; v < NV; ++v) d[(size_t)v * NCELL] = U[v];
    } else if (FINE && a.push_fine && n[q] <= -2 && n[q] != PUSH_BY_COARSER && (c[q] == 0 || c[q] == NI - 1)) {
      // finer neighbours (Q-G4, first order): the cell covers 2 x 2 x 2 ghost cells of one of them
      const int t0 = (q == 0) ? 1 : 0, t1 = (q == 2) ? 1 : 2;            // tangential axes, ascending
      const int nb = a.push_fine[(size_t)(-2 - n[q]) * 4 + (c[t0] >> 2) + 2 * (c[t1] >> 2)];
      int s[3];                                                         // storage index of the first fine ghost cell
      s[q] = (c[q] == 0) ? NG + NI : 0;                                 // our low face = their high ghosts
      s[t0] = NG + 2 * (c[t0] & 3);
      s[t1] = NG + 2 * (c[t1] & 3);
      double* __restrict__ d = push_base(a, nb) + (size_t)nb * BLOCK_DOUBLES + (s[2] * NS + s[1]) * NS + s[0];
#pragma unroll
      for (int v = 0; v < NV; ++v) {
        const double2 w = make_double2(U[v], U[v]);                     // x pairs: storage index even, 16-byte aligned
        double* __restrict__ dv = d + (size_t)v * NCELL;
#pragma unroll
        for (int z = 0; z < 2; ++z)
#pragma unroll
          for (int y = 0; y < 2; ++y) *reinterpret_cast<double2*>(dv + (z * NS + y) * NS) = w;
      }
    }
  }
}

__device__ __forceinline__ void push_cell(const StageArgs& a, double* __restrict__ o, const int n[3], int b, int i, int j, int k,
                                          const double U[NV]) {
  if (a.push_fine) push_cell_t<true>(a, o, n, b, i, j, k, U);
  else push_cell_t<false>(a, o, n, b, i, j, k, U);
}

// ---- launchers (each enqueues exactly one kernel on `st`) -------------------------
// stage 0: wave speeds only (initial dt, Q-T2); 1: out = base + dt/2 R(in); 2: out = base + dt R(in);
// 3: the single stage of the one-stage scheme (Q-U2): like 2 with in = base, local dt_c from this pass
cudaError_t launch_stage_general(int stage, const StageArgs& a, cudaStream_t st);
// fused shared-memory kernel for blocks without B0 split and body cells
cudaError_t launch_stage_fused(int stage, const StageArgs& a, cudaStream_t st);
bool stage_fused_supports(const StageArgs& a);
bool stage_fused_handles_body(const StageArgs& a);

// ghost fill (a1-a4) of one state buffer: plan-driven product kernel / message-driven reference kernel
// list: the destination blocks to fill (device, n_blocks entries), nullptr = blocks 0 .. n_blocks-1
// push_nbr (the table of batl_grid.hpp) != nullptr: only the face ghosts of faces without a pushing
// same-level neighbour are filled (the pass that follows a stage on the product path).
// prim: the buffer holds primitive variables (buffer B inside a two-stage step): restriction and fixed
// boundary states still act on the conserved variables (Q-G2) and are converted on the fly
// pass: 0 = every ghost cell; with second-order prolongation (Q-G4b) 1 = everything but the prolonged
// cells, 2 = the prolonged cells only (they read ghost cells of the coarse block that pass 1 wrote);
// beta: the limiter parameter of the prolongation slopes; owner / peer_state: sharded grids (batl.h), the
// source blocks of other ranks are read from their mapped buffers
cudaError_t launch_ghost_fill(double* state, const uint32_t* plan, const int32_t* plan_id, const int32_t* plan_src,
                              const double* bc_cons, const int32_t* list, int n_blocks, cudaStream_t st,
                              bool prim = false, double gamma = 0.0, const int32_t* push_nbr = nullptr,
                              int pass = 0, double beta = 2.0, const int32_t* owner = nullptr,
                              double* const* peer_state = nullptr);
// flux correction (Q-G6b) after a stage: one CTA per block that has faces bordering finer blocks
// (fc_group: first record and number of records of the block in fc_list, batl_grid.hpp)
cudaError_t launch_flux_correction(int stage, const StageArgs& a, const int32_t* fc_list, const int32_t* fc_group,
                                   int n_groups, cudaStream_t st);
cudaError_t launch_ghost_fill_msg(double* state, const batl_ghost_msg* msg, const int32_t* msg_start,
                                  const double* bc_cons, int n_blocks, cudaStream_t st);
// physical cells: compact [nB][8][8^3] <-> tiled [nB][8][12^3]
cudaError_t launch_scatter_phys(const double* compact, double* state, int n_blocks, cudaStream_t st);
cudaError_t launch_gather_phys(const double* state, double* compact, int n_blocks, cudaStream_t st);
// dt bookkeeping: mode 0 = start (dt <- dt_next or dt_fixed), 1 = end of a step (t += dt; dt <- dt_next)
cudaError_t launch_tick(DevScalars* sc, int mode, int dt_mode, double dt_fixed, cudaStream_t st);
cudaError_t launch_reset_scalars(DevScalars* sc, cudaStream_t st);

cudaError_t init_kernel_attributes();

}  // namespace batl
