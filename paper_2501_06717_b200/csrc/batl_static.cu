// mhd_stable_dt_static (include/batl.h): the CFL time step of a tiled state, for callers that cannot
// allocate -- code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
//
// It is the wave-speed pass of the step (stage 0 of stage_general_kernel: step a9, reading Q-T1 / Q-T2 of
// DESIGN.md; Alg. 1 L29-64 "calculate time step") run OUTSIDE a batl_grid.  Inside a grid that
// kernel keeps its working data in the caller-owned scratch buffer of batl_bind: the per-block geometry
// table and the device scalars that carry the running minimum and the warning bits.  Here the same data
// live in ONE file-scope device array of fixed size, so the call needs no buffer besides its inputs and
// outputs and calls neither cudaMalloc / cudaFree nor any allocating library routine.
//
// The array is shared by every call in the process (per device: each GPU that loads the library holds
// its own copy until exit) and keeps the last call's contents.  Every call rewrites the entries it reads
// (geometry of blocks 0 .. n_blocks-1, the scalars) in a kernel enqueued ahead of the reduction on the
// caller's stream, so calls on ONE stream are independent of one another; calls that overlap on the GPU
// (different streams, different host threads without ordering) race on it.
#include <mutex>
#include <string>

#include "batl.h"
#include "batl_device.cuh"

using namespace batl;

namespace {

constexpr int STATIC_MAX_BLOCKS = BATL_STATIC_MAX_BLOCKS;             // 4,096 blocks = 2,097,152 cells
constexpr size_t STATIC_OFF_GEOM = 256;                              // scalars first, then the geometry table
constexpr size_t STATIC_BYTES = STATIC_OFF_GEOM + (size_t)STATIC_MAX_BLOCKS * sizeof(BlockGeom);   // 360,704 B
static_assert(sizeof(DevScalars) <= STATIC_OFF_GEOM, "scalars do not fit their slot");
static_assert(sizeof(BlockGeom) % 8 == 0, "geometry table must keep doubles aligned");

// In host code this name is a host-side stand-in for the symbol, NOT a device address: the kernels get the
// address cudaGetSymbolAddress returns (static_scratch_of, below).
static __device__ __align__(256) unsigned char g_static_scratch[STATIC_BYTES];

constexpr int MAX_DEVICES = 64;
std::mutex g_mu;
unsigned char* g_scratch_ptr[MAX_DEVICES] = {};                      // per device, set once

thread_local std::string g_static_err;

// geometry rows and scalars of this call: what must start from a known value is written here every time
__global__ void static_prepare_kernel(const double* __restrict__ cell_size, int n_blocks, BlockGeom* __restrict__ geom,
                                      DevScalars* __restrict__ sc) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b == 0) {
    sc->dt = 0.0; sc->dt_last = 0.0; sc->t = 0.0;
    sc->dt_next_bits = 0x7FF0000000000000ull;                        // +inf: identity of the minimum
    sc->warn = 0; sc->pad = 0;
  }
  if (b >= n_blocks) return;
  BlockGeom G;
#pragma unroll
  for (int q = 0; q < 3; ++q) {
    const double D = cell_size[(size_t)b * 3 + q];
    G.x0[q] = 0.0;                                                   // positions enter only through B0 (not offered here)
    G.D[q] = D;
    G.invD[q] = 1.0 / D;                                             // correctly rounded: equal to the grid's 2^level / D_root
  }
  G.level = 0; G.flags = 0; G.mask_slot = -1; G.pad = 0;
  geom[b] = G;
}

__global__ void static_finish_kernel(const DevScalars* __restrict__ sc, double* __restrict__ dt, int32_t* __restrict__ warn) {
  *dt = __longlong_as_double((long long)sc->dt_next_bits);
  if (warn) *warn = sc->warn;
}

// Once per device, with that device current: the device address of the array, and the opt-in of the
// general stage kernel to its dynamic shared memory (batl_bind does the same for grids).
cudaError_t static_scratch_of(int dev, unsigned char** out) {
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_scratch_ptr[dev]) {
    unsigned char* p = nullptr;
    cudaError_t e = cudaGetSymbolAddress((void**)&p, g_static_scratch);
    if (e != cudaSuccess) return e;
    e = init_kernel_attributes();
    if (e != cudaSuccess) return e;
    g_scratch_ptr[dev] = p;
  }
  *out = g_scratch_ptr[dev];
  return cudaSuccess;
}

int static_fail(int code, const std::string& msg) {
  g_static_err = msg;
  return code;
}

}  // namespace

extern "C" const char* batl_static_last_error(void) { return g_static_err.c_str(); }

extern "C" int mhd_stable_dt_static(const double* d_tiles, const double* d_cell_size, int32_t n_blocks, double gamma,
                                    double cfl, double limiter_beta, int32_t n_order, int32_t flux_type,
                                    int32_t use_divb_source, double* d_dt, int32_t* d_warn, void* cuda_stream) {
  if (!d_tiles || !d_cell_size || !d_dt) return static_fail(BATL_EINVAL, "null argument");
  if (n_blocks < 1) return static_fail(BATL_EINVAL, "n_blocks must be at least 1");
  if (n_blocks > STATIC_MAX_BLOCKS)
    return static_fail(BATL_ENOMEM, "mhd_stable_dt_static: n_blocks = " + std::to_string(n_blocks) + " exceeds the " +
                                        std::to_string(STATIC_MAX_BLOCKS) + " blocks the static scratch array holds (" +
                                        std::to_string(STATIC_BYTES) + " bytes); bind a batl_grid for larger grids");
  if (((uintptr_t)d_tiles | (uintptr_t)d_cell_size | (uintptr_t)d_dt) & 7)
    return static_fail(BATL_EINVAL, "device pointers must be 8-byte aligned");
  if (!(gamma > 1.0) || !(cfl > 0.0)) return static_fail(BATL_EINVAL, "gamma must exceed 1 and cfl must be positive");
  if (n_order == 0) n_order = 2;
  if (n_order != 1 && n_order != 2) return static_fail(BATL_EINVAL, "n_order must be 1 or 2");
  if (flux_type != 0 && flux_type != 1) return static_fail(BATL_EINVAL, "flux_type must be 0 or 1");
  if (n_order == 2 && !(limiter_beta >= 1.0 && limiter_beta <= 2.0))
    return static_fail(BATL_EINVAL, "limiter_beta must lie in [1, 2]");

  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return static_fail(BATL_ECUDA, std::string("cudaGetDevice: ") + cudaGetErrorString(e));
  if (dev < 0 || dev >= MAX_DEVICES) return static_fail(BATL_EINVAL, "device ordinal beyond 63");
  unsigned char* scratch = nullptr;
  e = static_scratch_of(dev, &scratch);
  if (e != cudaSuccess) return static_fail(BATL_ECUDA, std::string("cudaGetSymbolAddress: ") + cudaGetErrorString(e));

  cudaStream_t st = (cudaStream_t)cuda_stream;
  DevScalars* sc = reinterpret_cast<DevScalars*>(scratch);
  BlockGeom* geom = reinterpret_cast<BlockGeom*>(scratch + STATIC_OFF_GEOM);

  static_prepare_kernel<<<(n_blocks + 127) / 128, 128, 0, st>>>(d_cell_size, n_blocks, geom, sc);
  e = cudaGetLastError();
  if (e != cudaSuccess) return static_fail(BATL_ECUDA, std::string("static_prepare_kernel: ") + cudaGetErrorString(e));

  StageArgs a;
  a.in = d_tiles; a.base = d_tiles; a.out = nullptr;                 // stage 0 reads `in` only and writes no state
  a.geom = geom;
  a.body_mask = nullptr;
  a.dt_local = nullptr;
  a.sc = sc;
  a.gamma = gamma; a.cfl = cfl; a.beta = (n_order == 1) ? 0.0 : limiter_beta;
  a.gm1 = gamma - 1.0; a.inv_gm1 = 1.0 / a.gm1; a.half_beta = 0.5 * a.beta;
  a.m[0] = a.m[1] = a.m[2] = 0.0;
  a.rho_body = 0.0; a.p_body = 0.0;
  a.dt_mode = BATL_DT_GLOBAL; a.use_divb = use_divb_source ? 1 : 0; a.use_b0 = 0; a.use_body = 0;
  a.n_order = n_order; a.flux_type = flux_type;
  a.b_prim = 0;
  a.n_blocks = n_blocks;
  a.n_sm = 0;
  a.blocks = nullptr; a.n_list = 0;
  a.push_nbr = nullptr; a.push_fine = nullptr;
  a.fc_slot = nullptr; a.fc_buf = nullptr;
  a.fused_body = 0;
  a.owner = nullptr; a.peer_out = nullptr; a.rank = 0;
  e = launch_stage_general(0, a, st);
  if (e != cudaSuccess) return static_fail(BATL_ECUDA, std::string("stage_general_kernel<0>: ") + cudaGetErrorString(e));

  static_finish_kernel<<<1, 1, 0, st>>>(sc, d_dt, d_warn);
  e = cudaGetLastError();
  if (e != cudaSuccess) return static_fail(BATL_ECUDA, std::string("static_finish_kernel: ") + cudaGetErrorString(e));
  return BATL_OK;
}
