// C ABI of include/batl.h.  Host bookkeeping only: every step of the hot path runs
// in the kernels of batl_kernels.cu / batl_stage_fused.cu.
#include <cstddef>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <utility>
#include <vector>

#include "batl.h"
#include "batl_device.cuh"

using namespace batl;

static thread_local std::string g_err;
static int fail(int code, const std::string& msg) { g_err = msg; return code; }
static int fail_cuda(cudaError_t e, const char* what) {
  g_err = std::string(what) + ": " + cudaGetErrorString(e);
  return BATL_ECUDA;
}
#define CU(call)                                              \
  do {                                                        \
    cudaError_t e__ = (call);                                 \
    if (e__ != cudaSuccess) return fail_cuda(e__, #call);     \
  } while (0)

static size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

// The tiles start STATE_SHIFT doubles into the caller's (256-byte aligned) state buffers: storage
// column 0 of every 12-double row then sits at byte 16 of a 32-byte DRAM sector, so the 8 physical
// cells of a row are two whole sectors -- the stage kernel's row stores, its U^n loads and the
// z-slab boxes of the tile are full-sector transfers -- and the ghost pair at the end of a row
// shares its sector with the ghost pair at the start of the next row.
static constexpr size_t STATE_SHIFT = 2;
static constexpr size_t STATE_PAD_BYTES = 256;

struct batl_grid {
  HostGrid h;
  // layout of the caller-owned scratch buffer
  size_t off_scalars = 0, off_geom = 0, off_msg_start = 0, off_msg = 0, off_mask = 0, off_bc = 0, off_dtl = 0;
  size_t off_plan = 0, off_plan_id = 0, off_plan_src = 0, off_lists = 0, off_push = 0, off_fill_list = 0;
  size_t off_prolong_list = 0, off_fc_slot = 0, off_fc_list = 0, off_fc_group = 0, off_fc_buf = 0;
  size_t scratch_bytes = 0, state_bytes = 0;
  // binding
  bool bound = false;
  double *A = nullptr, *B = nullptr;
  unsigned char* scratch = nullptr;
  cudaStream_t stream = nullptr;
  bool have_state = false;
  bool need_dt0 = true;          // global dt: stage-0 pass before the first step (Q-T2)
  bool ghost_full = false;       // every ghost cell of A is current (false after a step on the push path:
                                 // edge and corner ghosts of the blocks off the fill list are stale)
  int variant = 0;
  int n_sm = 0;                  // of the device current at batl_bind
  bool level_jumps = false;      // some block has a finer neighbour (restricted ghost cells exist)
  int64_t launches = 0;
  int64_t n_fused = 0, n_general = 0, n_general_fallback = 0, n_fill = 0, n_fill_blocks = 0;
  // opt-in phase timers
  bool timers = false;
  double ms_stage = 0, ms_ghost = 0, ms_other = 0;
  struct Span { cudaEvent_t a, b; int phase; bool closed; };
  std::vector<Span> spans;
  std::vector<cudaEvent_t> event_pool;

  DevScalars* d_scalars() const { return reinterpret_cast<DevScalars*>(scratch + off_scalars); }
  BlockGeom* d_geom() const { return reinterpret_cast<BlockGeom*>(scratch + off_geom); }
  int32_t* d_msg_start() const { return reinterpret_cast<int32_t*>(scratch + off_msg_start); }
  batl_ghost_msg* d_msg() const { return reinterpret_cast<batl_ghost_msg*>(scratch + off_msg); }
  uint32_t* d_mask() const { return reinterpret_cast<uint32_t*>(scratch + off_mask); }
  double* d_bc() const { return reinterpret_cast<double*>(scratch + off_bc); }
  double* d_dtl() const { return reinterpret_cast<double*>(scratch + off_dtl); }
  uint32_t* d_plan() const { return reinterpret_cast<uint32_t*>(scratch + off_plan); }
  int32_t* d_plan_id() const { return reinterpret_cast<int32_t*>(scratch + off_plan_id); }
  int32_t* d_plan_src() const { return reinterpret_cast<int32_t*>(scratch + off_plan_src); }
  int32_t* d_list_plain() const { return reinterpret_cast<int32_t*>(scratch + off_lists); }
  int32_t* d_list_body() const { return d_list_plain() + l_plain().size(); }
  int32_t* d_push() const { return reinterpret_cast<int32_t*>(scratch + off_push); }
  int32_t* d_fill_list() const { return reinterpret_cast<int32_t*>(scratch + off_fill_list); }
  int32_t* d_prolong_list() const { return reinterpret_cast<int32_t*>(scratch + off_prolong_list); }
  int32_t* d_fc_slot() const { return reinterpret_cast<int32_t*>(scratch + off_fc_slot); }
  int32_t* d_fc_list() const { return reinterpret_cast<int32_t*>(scratch + off_fc_list); }
  int32_t* d_fc_group() const { return reinterpret_cast<int32_t*>(scratch + off_fc_group); }
  double* d_fc_buf() const { return reinterpret_cast<double*>(scratch + off_fc_buf); }
  int64_t n_flux_corr = 0;
  // sharding (batl_set_partition): contiguous Morton segments; lists filtered to the own blocks
  int world = 1, rank = 0;
  std::vector<int32_t> first_block, owner;
  std::vector<int32_t> own_all, own_plain, own_body, own_fill;
  size_t off_owner = 0, off_own_all = 0, off_peers = 0, off_push_fine = 0;
  int32_t* d_push_fine() const { return reinterpret_cast<int32_t*>(scratch + off_push_fine); }
  bool peers_bound = false;
  double* A_bound = nullptr;     // buffer A as given to batl_bind: the peer tables are indexed by buffer, not by role
  int32_t* d_owner() const { return reinterpret_cast<int32_t*>(scratch + off_owner); }
  int32_t* d_own_all() const { return reinterpret_cast<int32_t*>(scratch + off_own_all); }
  double** d_peerA() const { return reinterpret_cast<double**>(scratch + off_peers); }
  double** d_peerB() const { return d_peerA() + 64; }
  bool sharded() const { return world > 1; }
  const std::vector<int32_t>& l_plain() const { return sharded() ? own_plain : h.list_plain; }
  const std::vector<int32_t>& l_body() const { return sharded() ? own_body : h.list_body; }
  const std::vector<int32_t>& l_fill() const { return sharded() ? own_fill : h.list_fill; }
};

extern "C" {

const char* batl_last_error(void) { return g_err.c_str(); }

int batl_init_grid(const batl_config* cfg, batl_grid** out) {
  if (!cfg || !out) return fail(BATL_EINVAL, "null argument");
  *out = nullptr;
  batl_grid* g = new (std::nothrow) batl_grid();
  if (!g) return fail(BATL_ENOMEM, "out of host memory");
  std::string err;
  int rc;
  try {
    rc = build_grid(*cfg, g->h, err);
  } catch (const std::bad_alloc&) {
    delete g;
    return fail(BATL_ENOMEM, "out of host memory");
  }
  if (rc != BATL_OK) { delete g; return fail(rc, err); }
  const size_t nB = (size_t)g->h.n_blocks();
  for (int8_t d : g->h.dlev) if (d == -1) { g->level_jumps = true; break; }
  size_t o = 0;
  g->off_scalars = o;   o = align256(o + sizeof(DevScalars));
  g->off_geom = o;      o = align256(o + nB * sizeof(BlockGeom));
  g->off_msg_start = o; o = align256(o + (nB + 1) * sizeof(int32_t));
  g->off_msg = o;       o = align256(o + g->h.msg.size() * sizeof(batl_ghost_msg));
  g->off_mask = o;      o = align256(o + g->h.body_mask.size() * sizeof(uint32_t));
  g->off_bc = o;        o = align256(o + 12 * NV * sizeof(double));   // fixed boundary states: conserved, then primitive
  g->off_plan = o;      o = align256(o + g->h.plan.size() * sizeof(uint32_t));
  g->off_plan_id = o;   o = align256(o + nB * sizeof(int32_t));
  g->off_plan_src = o;  o = align256(o + g->h.plan_src.size() * sizeof(int32_t));
  g->off_lists = o;     o = align256(o + nB * sizeof(int32_t));
  g->off_push = o;      o = align256(o + nB * 6 * sizeof(int32_t));
  g->off_fill_list = o; o = align256(o + nB * sizeof(int32_t));
  g->off_prolong_list = o; o = align256(o + nB * sizeof(int32_t));
  g->off_fc_slot = o;   o = align256(o + nB * 6 * sizeof(int32_t));
  g->off_fc_list = o;   o = align256(o + g->h.fc_list.size() * sizeof(int32_t));
  g->off_fc_group = o;  o = align256(o + g->h.fc_group.size() * sizeof(int32_t));
  g->off_fc_buf = o;    o = align256(o + (size_t)g->h.n_fc_slots * NV * NI * NI * sizeof(double));
  g->off_push_fine = o; o = align256(o + g->h.push_fine.size() * sizeof(int32_t));
  g->off_owner = o;     o = align256(o + nB * sizeof(int32_t));
  g->off_own_all = o;   o = align256(o + nB * sizeof(int32_t));
  g->off_peers = o;     o = align256(o + 2 * 64 * sizeof(double*));   // up to 64 ranks: mapped A and B buffers
  g->off_dtl = o;
  if (cfg->dt_mode == BATL_DT_LOCAL) o = align256(o + nB * NPHYS * sizeof(double));
  g->scratch_bytes = o;
  g->state_bytes = nB * BLOCK_BYTES + STATE_PAD_BYTES;
  *out = g;
  return BATL_OK;
}

void batl_free_grid(batl_grid* g) {
  if (!g) return;
  for (auto& s : g->spans) { cudaEventDestroy(s.a); cudaEventDestroy(s.b); }
  for (auto e : g->event_pool) cudaEventDestroy(e);
  delete g;
}

int batl_n_blocks(const batl_grid* g, int32_t* n) {
  if (!g || !n) return fail(BATL_EINVAL, "null argument");
  *n = g->h.n_blocks();
  return BATL_OK;
}

int batl_buffer_bytes(const batl_grid* g, size_t* state_bytes, size_t* scratch_bytes) {
  if (!g) return fail(BATL_EINVAL, "null argument");
  if (state_bytes) *state_bytes = g->state_bytes;
  if (scratch_bytes) *scratch_bytes = g->scratch_bytes;
  return BATL_OK;
}

int batl_get_blocks(const batl_grid* g, int32_t* out) {
  if (!g || !out) return fail(BATL_EINVAL, "null argument");
  for (int b = 0; b < g->h.n_blocks(); ++b) {
    out[4 * b] = g->h.leaf[b].level;
    for (int a = 0; a < 3; ++a) out[4 * b + 1 + a] = g->h.leaf[b].I[a];
  }
  return BATL_OK;
}

int batl_get_neighbors(const batl_grid* g, int32_t* nbr, int8_t* dlev) {
  if (!g) return fail(BATL_EINVAL, "null argument");
  if (nbr) std::memcpy(nbr, g->h.nbr.data(), g->h.nbr.size() * sizeof(int32_t));
  if (dlev) std::memcpy(dlev, g->h.dlev.data(), g->h.dlev.size());
  return BATL_OK;
}

int batl_get_ghost_list(const batl_grid* g, int32_t kind, void* out, size_t* n) {
  if (!g || !n) return fail(BATL_EINVAL, "null argument");
  if (kind == BATL_LIST_MESSAGES) {
    *n = g->h.msg.size();
    if (out) std::memcpy(out, g->h.msg.data(), g->h.msg.size() * sizeof(batl_ghost_msg));
    return BATL_OK;
  }
  if (kind == BATL_LIST_EXPANDED) {
    *n = (size_t)g->h.n_blocks() * (NCELL - NPHYS);
    if (out) {
      std::vector<int32_t> rows;
      expand_ghost_list(g->h, rows);
      if (rows.size() != *n * 9) return fail(BATL_EGRID, "ghost messages do not cover every ghost cell exactly once");
      std::memcpy(out, rows.data(), rows.size() * sizeof(int32_t));
    }
    return BATL_OK;
  }
  if (kind == BATL_LIST_PLAN) {
    *n = (size_t)g->h.n_blocks() * NGHOST;
    if (out) {
      std::vector<int32_t> rows;
      expand_plan_list(g->h, rows);
      std::memcpy(out, rows.data(), rows.size() * sizeof(int32_t));
    }
    return BATL_OK;
  }
  if (kind == BATL_LIST_PLAN_PATTERNS) {
    *n = g->h.plan.size() / NGHOST;
    if (out) std::memcpy(out, g->h.plan.data(), g->h.plan.size() * sizeof(uint32_t));
    return BATL_OK;
  }
  if (kind == BATL_LIST_PLAN_IDS) {
    *n = g->h.plan_id.size();
    if (out) std::memcpy(out, g->h.plan_id.data(), g->h.plan_id.size() * sizeof(int32_t));
    return BATL_OK;
  }
  if (kind == BATL_LIST_FC_SLOTS) {
    *n = g->h.fc_slot.size() / 6;
    if (out) std::memcpy(out, g->h.fc_slot.data(), g->h.fc_slot.size() * sizeof(int32_t));
    return BATL_OK;
  }
  if (kind == BATL_LIST_FC_RECORDS) {
    *n = g->h.fc_list.size() / 8;
    if (out && !g->h.fc_list.empty()) std::memcpy(out, g->h.fc_list.data(), g->h.fc_list.size() * sizeof(int32_t));
    return BATL_OK;
  }
  return fail(BATL_EINVAL, "unknown ghost list kind");
}

int batl_bind(batl_grid* g, void* d_stateA, void* d_stateB, void* d_scratch, void* cuda_stream) {
  if (!g || !d_stateA || !d_stateB || !d_scratch) return fail(BATL_EINVAL, "null argument");
  if (((uintptr_t)d_stateA | (uintptr_t)d_stateB | (uintptr_t)d_scratch) & 255)
    return fail(BATL_EINVAL, "device buffers must be 256-byte aligned");
  int ndev = 0;
  CU(cudaGetDeviceCount(&ndev));
  if (ndev == 0) return fail(BATL_ECUDA, "no CUDA device");
  CU(init_kernel_attributes());
  int dev = 0;
  CU(cudaGetDevice(&dev));
  CU(cudaDeviceGetAttribute(&g->n_sm, cudaDevAttrMultiProcessorCount, dev));
  g->A = (double*)d_stateA + STATE_SHIFT;
  g->B = (double*)d_stateB + STATE_SHIFT;
  g->A_bound = g->A;
  g->scratch = (unsigned char*)d_scratch;
  g->stream = (cudaStream_t)cuda_stream;
  cudaStream_t st = g->stream;
  const HostGrid& h = g->h;
  CU(cudaMemcpyAsync(g->d_geom(), h.geom.data(), h.geom.size() * sizeof(BlockGeom), cudaMemcpyHostToDevice, st));
  CU(cudaMemcpyAsync(g->d_msg_start(), h.msg_start.data(), h.msg_start.size() * sizeof(int32_t), cudaMemcpyHostToDevice, st));
  if (!h.msg.empty())
    CU(cudaMemcpyAsync(g->d_msg(), h.msg.data(), h.msg.size() * sizeof(batl_ghost_msg), cudaMemcpyHostToDevice, st));
  if (!h.body_mask.empty())
    CU(cudaMemcpyAsync(g->d_mask(), h.body_mask.data(), h.body_mask.size() * sizeof(uint32_t), cudaMemcpyHostToDevice, st));
  CU(cudaMemcpyAsync(g->d_bc(), &h.bc_cons[0][0], 6 * NV * sizeof(double), cudaMemcpyHostToDevice, st));
  CU(cudaMemcpyAsync(g->d_bc() + 6 * NV, &h.cfg.bc_prim[0][0], 6 * NV * sizeof(double), cudaMemcpyHostToDevice, st));
  if (!h.plan.empty()) {
    CU(cudaMemcpyAsync(g->d_plan(), h.plan.data(), h.plan.size() * sizeof(uint32_t), cudaMemcpyHostToDevice, st));
    CU(cudaMemcpyAsync(g->d_plan_id(), h.plan_id.data(), h.plan_id.size() * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    CU(cudaMemcpyAsync(g->d_plan_src(), h.plan_src.data(), h.plan_src.size() * sizeof(int32_t), cudaMemcpyHostToDevice, st));
  }
  if (!g->l_plain().empty())
    CU(cudaMemcpyAsync(g->d_list_plain(), g->l_plain().data(), g->l_plain().size() * sizeof(int32_t), cudaMemcpyHostToDevice, st));
  if (!g->l_body().empty())
    CU(cudaMemcpyAsync(g->d_list_body(), g->l_body().data(), g->l_body().size() * sizeof(int32_t), cudaMemcpyHostToDevice, st));
  if (g->sharded()) {
    CU(cudaMemcpyAsync(g->d_owner(), g->owner.data(), g->owner.size() * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    CU(cudaMemcpyAsync(g->d_own_all(), g->own_all.data(), g->own_all.size() * sizeof(int32_t), cudaMemcpyHostToDevice, st));
  }
  g->peers_bound = false;
  CU(cudaMemcpyAsync(g->d_push(), h.push_nbr.data(), h.push_nbr.size() * sizeof(int32_t), cudaMemcpyHostToDevice, st));
  if (!h.push_fine.empty())
    CU(cudaMemcpyAsync(g->d_push_fine(), h.push_fine.data(), h.push_fine.size() * sizeof(int32_t), cudaMemcpyHostToDevice, st));
  if (!g->l_fill().empty())
    CU(cudaMemcpyAsync(g->d_fill_list(), g->l_fill().data(), g->l_fill().size() * sizeof(int32_t), cudaMemcpyHostToDevice, st));
  if (!h.list_prolong.empty())
    CU(cudaMemcpyAsync(g->d_prolong_list(), h.list_prolong.data(), h.list_prolong.size() * sizeof(int32_t), cudaMemcpyHostToDevice, st));
  CU(cudaMemcpyAsync(g->d_fc_slot(), h.fc_slot.data(), h.fc_slot.size() * sizeof(int32_t), cudaMemcpyHostToDevice, st));
  if (!h.fc_list.empty()) {
    CU(cudaMemcpyAsync(g->d_fc_list(), h.fc_list.data(), h.fc_list.size() * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    CU(cudaMemcpyAsync(g->d_fc_group(), h.fc_group.data(), h.fc_group.size() * sizeof(int32_t), cudaMemcpyHostToDevice, st));
  }
  CU(launch_reset_scalars(g->d_scalars(), st));
  g->launches = 1;
  CU(cudaStreamSynchronize(st));        // the host tables may go away after this call
  g->bound = true;
  g->have_state = false;
  g->need_dt0 = true;
  return BATL_OK;
}

// ---- phase timers ------------------------------------------------------------------
// Two events per launch, taken from a pool and returned to it when collected; the spans are
// collected whenever MAX_SPANS are pending (mhd_step_async(n) with a large n), so the list
// stays bounded.  A span whose end was never recorded (a launch failed in between) is dropped.
static constexpr size_t MAX_SPANS = 4096;
static void spans_collect(batl_grid* g);
static cudaEvent_t event_from_pool(batl_grid* g) {
  cudaEvent_t e = nullptr;
  if (!g->event_pool.empty()) { e = g->event_pool.back(); g->event_pool.pop_back(); return e; }
  return cudaEventCreate(&e) == cudaSuccess ? e : nullptr;
}
static void span_begin(batl_grid* g, int phase) {
  if (!g->timers) return;
  if (g->spans.size() >= MAX_SPANS) spans_collect(g);
  batl_grid::Span s;
  s.a = event_from_pool(g);
  s.b = event_from_pool(g);
  s.phase = phase;
  s.closed = false;
  if (!s.a || !s.b || cudaEventRecord(s.a, g->stream) != cudaSuccess) {
    if (s.a) g->event_pool.push_back(s.a);
    if (s.b) g->event_pool.push_back(s.b);
    return;                                  // no span: span_end finds none open
  }
  g->spans.push_back(s);
}
static void span_end(batl_grid* g) {
  if (!g->timers || g->spans.empty() || g->spans.back().closed) return;
  g->spans.back().closed = cudaEventRecord(g->spans.back().b, g->stream) == cudaSuccess;
}
static void spans_collect(batl_grid* g) {
  for (auto& s : g->spans) {
    float ms = 0.f;
    if (s.closed && cudaEventSynchronize(s.b) == cudaSuccess && cudaEventElapsedTime(&ms, s.a, s.b) == cudaSuccess)
      (s.phase == 0 ? g->ms_stage : s.phase == 1 ? g->ms_ghost : g->ms_other) += ms;
    g->event_pool.push_back(s.a);
    g->event_pool.push_back(s.b);
  }
  g->spans.clear();
}

static bool b_holds_primitives(const batl_grid* g) {
  const batl_config& c = g->h.cfg;
  // measured (B200): on grids with resolution changes the restriction of a primitive buffer (conserved means,
  // three conversions per restricted ghost cell) costs more than the conversion pass it saves (config 5
  // 0.786 -> 0.764, config 3 0.097 -> 0.089 ms/step with B conserved), so only single-level grids use it
  return g->variant == 0 && c.n_stage == 2 && c.prolong_order == 1 && !c.flux_correction && !g->level_jumps;
}

static StageArgs stage_args(const batl_grid* g, const double* in, const double* base, double* out) {
  StageArgs a;
  const batl_config& c = g->h.cfg;
  a.in = in; a.base = base; a.out = out;
  a.geom = g->d_geom();
  a.body_mask = g->d_mask();
  a.dt_local = (c.dt_mode == BATL_DT_LOCAL) ? g->d_dtl() : nullptr;
  a.sc = g->d_scalars();
  // n_order = 1 (piecewise-constant face states): beta = 0 makes every limited slope exactly +-0
  a.gamma = c.gamma; a.cfl = c.cfl; a.beta = (c.n_order == 1) ? 0.0 : c.limiter_beta;
  a.gm1 = c.gamma - 1.0; a.inv_gm1 = 1.0 / a.gm1; a.half_beta = 0.5 * a.beta;
  for (int q = 0; q < 3; ++q) a.m[q] = c.dipole_m[q];
  a.rho_body = c.rho_body; a.p_body = c.p_body;
  a.dt_mode = c.dt_mode; a.use_divb = c.use_divb_source; a.use_b0 = c.use_b0; a.use_body = c.use_body;
  a.n_order = c.n_order; a.flux_type = c.flux_type;
  a.n_blocks = g->h.n_blocks();
  a.n_sm = g->n_sm;
  a.blocks = nullptr; a.n_list = 0;
  // product path: the stage kernels write their outer cell layers into the neighbours' face ghosts
  a.push_nbr = (g->variant == 0) ? g->d_push() : nullptr;
  a.push_fine = g->h.push_fine.empty() ? nullptr : g->d_push_fine();
  // product path: U* (buffer B) travels between the two stages as primitive variables, unless an
  // operator at resolution changes needs it conserved (second-order prolongation, flux correction)
  a.b_prim = b_holds_primitives(g) ? 1 : 0;
  const bool fc = c.flux_correction && !g->h.fc_list.empty();
  a.fc_slot = fc ? g->d_fc_slot() : nullptr;
  a.fc_buf = fc ? g->d_fc_buf() : nullptr;
  a.fused_body = 0;
  a.owner = nullptr; a.peer_out = nullptr; a.rank = 0;
  return a;
}

static int enqueue_stage(batl_grid* g, int stage, const double* in, const double* base, double* out) {
  StageArgs a = stage_args(g, in, base, out);
  if (g->sharded()) {                                      // pushes into blocks of other ranks go through their buffers
    a.owner = g->d_owner();
    a.rank = g->rank;
    a.peer_out = (out == g->A_bound) ? g->d_peerA() : g->d_peerB();
  }
  span_begin(g, 0);
  cudaError_t e = cudaSuccess;
  if (g->sharded()) {                                      // own blocks only: fused kernel on the body-free ones, general on the rest
    a.blocks = g->d_list_plain(); a.n_list = (int)g->own_plain.size();
    if (a.n_list > 0) { e = launch_stage_fused(stage, a, g->stream); g->launches++; g->n_fused++; }
    if (e == cudaSuccess && !g->own_body.empty()) {
      a.blocks = g->d_list_body(); a.n_list = (int)g->own_body.size();
      e = launch_stage_general(stage, a, g->stream);
      g->launches++; g->n_general++;
    }
  } else if (g->variant != 0 || !stage_fused_supports(a)) {     // reference path: general kernel on every block
    e = launch_stage_general(stage, a, g->stream);
    g->launches++; g->n_general++;
    if (g->variant == 0) g->n_general_fallback++;        // not asked for: the fused kernel lacks this combination
  } else if (g->h.list_body.empty() || stage_fused_handles_body(a)) {   // fused kernel on every block
    a.fused_body = g->h.list_body.empty() ? 0 : 1;
    e = launch_stage_fused(stage, a, g->stream);
    g->launches++; g->n_fused++;
  } else {                                               // fused kernel on the body-free blocks, general on the rest
    a.blocks = g->d_list_plain(); a.n_list = (int)g->h.list_plain.size();
    if (a.n_list > 0) { e = launch_stage_fused(stage, a, g->stream); g->launches++; g->n_fused++; }
    if (e == cudaSuccess) {
      a.blocks = g->d_list_body(); a.n_list = (int)g->h.list_body.size();
      e = launch_stage_general(stage, a, g->stream);
      g->launches++; g->n_general++;
    }
  }
  if (e == cudaSuccess && stage != 0 && a.fc_slot) {      // Q-G6b: coarse cells next to finer blocks take the fine fluxes
    a.blocks = nullptr; a.n_list = 0;
    e = launch_flux_correction(stage, a, g->d_fc_list(), g->d_fc_group(), (int)(g->h.fc_group.size() / 2), g->stream);
    g->launches++; g->n_flux_corr++;
  }
  span_end(g);
  CU(e);
  return BATL_OK;
}

// full = 1: every ghost cell of every block (after set_state, on request, reference path).
// full = 0, product path: the stage kernel has already pushed the same-level face ghosts, so only
// the faces at resolution changes and boundaries of the blocks of list_fill are filled -- none on a
// uniform periodic grid, where this enqueues nothing.
static int enqueue_fill(batl_grid* g, double* S, bool full, bool prim = false) {
  const int nB = g->h.n_blocks();
  const batl_config& c = g->h.cfg;
  const double gamma = c.gamma, beta = c.limiter_beta;
  // second-order prolongation (Q-G4b): copy / restriction / boundary states first, then the prolonged
  // cells of the blocks that have some (they read ghost cells of the coarser block)
  const bool two = c.prolong_order == 2 && !g->h.list_prolong.empty();
  const int n_pro = (int)g->h.list_prolong.size();
  cudaError_t e = cudaSuccess;
  if (g->variant != 0 && two) full = true;                // the message-walking reference kernel is first order only
  if (g->variant != 0 && !two) {
    span_begin(g, 1);
    e = launch_ghost_fill_msg(S, g->d_msg(), g->d_msg_start(), g->d_bc(), nB, g->stream);
    span_end(g);
    g->launches++; g->n_fill++; g->n_fill_blocks += nB;
  } else if (full) {
    span_begin(g, 1);
    e = launch_ghost_fill(S, g->d_plan(), g->d_plan_id(), g->d_plan_src(), g->d_bc(), nullptr, nB, g->stream, prim, gamma,
                          nullptr, two ? 1 : 0, beta);
    g->launches++; g->n_fill++; g->n_fill_blocks += nB;
    if (e == cudaSuccess && two) {
      e = launch_ghost_fill(S, g->d_plan(), g->d_plan_id(), g->d_plan_src(), g->d_bc(), g->d_prolong_list(), n_pro, g->stream,
                            prim, gamma, nullptr, 2, beta);
      g->launches++; g->n_fill++; g->n_fill_blocks += n_pro;
    }
    span_end(g);
  } else if (!g->l_fill().empty()) {
    const int n = (int)g->l_fill().size();
    span_begin(g, 1);
    e = launch_ghost_fill(S, g->d_plan(), g->d_plan_id(), g->d_plan_src(), g->d_bc(), g->d_fill_list(), n, g->stream, prim, gamma,
                          g->d_push(), two ? 1 : 0, beta, g->sharded() ? g->d_owner() : nullptr,
                          g->sharded() ? (S == g->A_bound ? g->d_peerA() : g->d_peerB()) : nullptr);
    g->launches++; g->n_fill++; g->n_fill_blocks += n;
    if (e == cudaSuccess && two) {
      e = launch_ghost_fill(S, g->d_plan(), g->d_plan_id(), g->d_plan_src(), g->d_bc(), g->d_prolong_list(), n_pro, g->stream,
                            prim, gamma, g->d_push(), 2, beta);
      g->launches++; g->n_fill++; g->n_fill_blocks += n_pro;
    }
    span_end(g);
  }
  CU(e);
  return BATL_OK;
}

static int enqueue_tick(batl_grid* g, int mode) {
  span_begin(g, 2);
  CU(launch_tick(g->d_scalars(), mode, g->h.cfg.dt_mode, g->h.cfg.dt_fixed, g->stream));
  span_end(g);
  g->launches++;
  return BATL_OK;
}

static int finish_set_state(batl_grid* g) {
  int rc;
  CU(launch_scatter_phys(g->B, g->A, g->h.n_blocks(), g->stream));
  g->launches++;
  if ((rc = enqueue_fill(g, g->A, true)) != BATL_OK) return rc;
  CU(launch_reset_scalars(g->d_scalars(), g->stream));
  g->launches++;
  g->have_state = true;
  g->need_dt0 = true;
  g->ghost_full = true;
  return BATL_OK;
}

int batl_set_state(batl_grid* g, const double* h_U) {
  if (!g || !h_U) return fail(BATL_EINVAL, "null argument");
  if (!g->bound) return fail(BATL_ENOTBOUND, "batl_bind has not been called");
  // buffer B is free between steps: use it as the staging area of the compact array
  CU(cudaMemcpyAsync(g->B, h_U, (size_t)g->h.n_blocks() * NV * NPHYS * sizeof(double), cudaMemcpyHostToDevice, g->stream));
  int rc = finish_set_state(g);
  if (rc != BATL_OK) return rc;
  CU(cudaStreamSynchronize(g->stream));   // h_U may be pageable: do not return before it has been read
  return BATL_OK;
}

int batl_set_state_device(batl_grid* g, const double* d_U) {
  if (!g || !d_U) return fail(BATL_EINVAL, "null argument");
  if (!g->bound) return fail(BATL_ENOTBOUND, "batl_bind has not been called");
  CU(cudaMemcpyAsync(g->B, d_U, (size_t)g->h.n_blocks() * NV * NPHYS * sizeof(double), cudaMemcpyDeviceToDevice, g->stream));
  return finish_set_state(g);
}

int batl_fill_ghosts(batl_grid* g) {
  if (!g) return fail(BATL_EINVAL, "null argument");
  if (!g->bound) return fail(BATL_ENOTBOUND, "batl_bind has not been called");
  const int rc = enqueue_fill(g, g->A, true);
  if (rc == BATL_OK) g->ghost_full = true;
  return rc;
}

// ---- sharding over the GPUs of one node (batl.h) -------------------------------------------------
int batl_set_partition(batl_grid* g, int32_t world, int32_t rank) {
  if (!g || world < 1 || world > 64 || rank < 0 || rank >= world) return fail(BATL_EINVAL, "bad world / rank (1 <= world <= 64)");
  if (g->bound) return fail(BATL_EINVAL, "batl_set_partition must precede batl_bind");
  const batl_config& c = g->h.cfg;
  if (world > 1 && (c.prolong_order != 1 || c.flux_correction))
    return fail(BATL_EINVAL, "sharded grids support first-order prolongation and no flux correction");
  const int nB = g->h.n_blocks();
  g->world = world; g->rank = rank;
  g->first_block.assign(world + 1, 0);
  for (int r = 0; r <= world; ++r) g->first_block[r] = (int32_t)((int64_t)nB * r / world);   // equal block counts (L117)
  g->owner.assign(nB, 0);
  for (int r = 0; r < world; ++r)
    for (int b = g->first_block[r]; b < g->first_block[r + 1]; ++b) g->owner[b] = r;
  auto mine = [&](const std::vector<int32_t>& in, std::vector<int32_t>& out) {
    out.clear();
    for (int32_t b : in) if (g->owner[b] == rank) out.push_back(b);
  };
  g->own_all.clear();
  for (int b = g->first_block[rank]; b < g->first_block[rank + 1]; ++b) g->own_all.push_back(b);
  mine(g->h.list_plain, g->own_plain);
  mine(g->h.list_body, g->own_body);
  mine(g->h.list_fill, g->own_fill);
  return BATL_OK;
}

int batl_get_partition(const batl_grid* g, int32_t* first_block) {
  if (!g || !first_block) return fail(BATL_EINVAL, "null argument");
  if (g->first_block.empty()) { first_block[0] = 0; first_block[1] = g->h.n_blocks(); return BATL_OK; }
  for (size_t r = 0; r < g->first_block.size(); ++r) first_block[r] = g->first_block[r];
  return BATL_OK;
}

int batl_bind_peers(batl_grid* g, void* const* d_stateA, void* const* d_stateB) {
  if (!g || !d_stateA || !d_stateB) return fail(BATL_EINVAL, "null argument");
  if (!g->bound) return fail(BATL_ENOTBOUND, "batl_bind has not been called");
  double* pa[64];
  double* pb[64];
  for (int r = 0; r < g->world; ++r) {
    if (!d_stateA[r] || !d_stateB[r]) return fail(BATL_EINVAL, "null peer buffer");
    pa[r] = (double*)d_stateA[r] + STATE_SHIFT;
    pb[r] = (double*)d_stateB[r] + STATE_SHIFT;
  }
  // the buffers may have traded roles (one-stage scheme) but never do on a sharded grid
  if (pa[g->rank] != g->A_bound || (pb[g->rank] != g->A && pb[g->rank] != g->B))
    return fail(BATL_EINVAL, "entry `rank` must be the buffers given to batl_bind");
  CU(cudaMemcpyAsync(g->d_peerA(), pa, g->world * sizeof(double*), cudaMemcpyHostToDevice, g->stream));
  CU(cudaMemcpyAsync(g->d_peerB(), pb, g->world * sizeof(double*), cudaMemcpyHostToDevice, g->stream));
  CU(cudaStreamSynchronize(g->stream));
  g->peers_bound = true;
  return BATL_OK;
}

int batl_scalar_offsets(const batl_grid* g, size_t* dt_next_offset) {
  if (!g || !dt_next_offset) return fail(BATL_EINVAL, "null argument");
  *dt_next_offset = g->off_scalars + offsetof(DevScalars, dt_next_bits);
  return BATL_OK;
}

int batl_step_part(batl_grid* g, int32_t part) {
  if (!g) return fail(BATL_EINVAL, "null argument");
  if (!g->bound) return fail(BATL_ENOTBOUND, "batl_bind has not been called");
  if (!g->have_state) return fail(BATL_EINVAL, "batl_set_state has not been called");
  if (g->sharded() && !g->peers_bound) return fail(BATL_ENOTBOUND, "batl_bind_peers has not been called");
  if (g->variant != 0) return fail(BATL_EINVAL, "batl_step_part: kernel variant 0 only");
  if (g->h.cfg.n_stage == 1) {                  // Q-U2: STAGE1 = the single stage (A -> B), FILL_B, TICK_END trades the buffers
    switch (part) {
      case BATL_PART_DT0:
        if (g->h.cfg.dt_mode == BATL_DT_GLOBAL) return enqueue_stage(g, 0, g->A, g->A, g->B);
        return BATL_OK;
      case BATL_PART_TICK_START: g->need_dt0 = false; return enqueue_tick(g, 0);
      case BATL_PART_STAGE1: g->ghost_full = false; return enqueue_stage(g, 3, g->A, g->A, g->B);
      case BATL_PART_FILL_B: return enqueue_fill(g, g->B, false);
      case BATL_PART_STAGE2: case BATL_PART_FILL_A: return BATL_OK;
      case BATL_PART_TICK_END: std::swap(g->A, g->B); return enqueue_tick(g, 1);
    }
    return fail(BATL_EINVAL, "unknown part");
  }
  switch (part) {
    case BATL_PART_DT0:
      if (g->h.cfg.dt_mode == BATL_DT_GLOBAL) return enqueue_stage(g, 0, g->A, g->A, g->B);
      return BATL_OK;
    case BATL_PART_TICK_START: g->need_dt0 = false; return enqueue_tick(g, 0);
    case BATL_PART_STAGE1: g->ghost_full = false; return enqueue_stage(g, 1, g->A, g->A, g->B);
    case BATL_PART_FILL_B: return enqueue_fill(g, g->B, false, b_holds_primitives(g));
    case BATL_PART_STAGE2: return enqueue_stage(g, 2, g->B, g->A, g->A);
    case BATL_PART_FILL_A: return enqueue_fill(g, g->A, false);
    case BATL_PART_TICK_END: return enqueue_tick(g, 1);
  }
  return fail(BATL_EINVAL, "unknown part");
}

int mhd_step_async(batl_grid* g, int32_t n_steps) {
  if (!g || n_steps < 0) return fail(BATL_EINVAL, "bad argument");
  if (!g->bound) return fail(BATL_ENOTBOUND, "batl_bind has not been called");
  if (!g->have_state) return fail(BATL_EINVAL, "batl_set_state has not been called");
  if (g->sharded() && n_steps > 0)
    return fail(BATL_EINVAL, "sharded grid: drive the step with batl_step_part (the ranks synchronise between the parts)");
  int rc;
  if (n_steps > 0 && g->variant == 0) g->ghost_full = false;   // product path: only face ghosts are kept current
  for (int s = 0; s < n_steps; ++s) {
    if (g->need_dt0) {                       // dt of the first step (Q-T2): speeds of the initial state
      if (g->h.cfg.dt_mode == BATL_DT_GLOBAL)
        if ((rc = enqueue_stage(g, 0, g->A, g->A, g->B)) != BATL_OK) return rc;
      if ((rc = enqueue_tick(g, 0)) != BATL_OK) return rc;
      g->need_dt0 = false;
    }
    if (g->h.cfg.n_stage == 1) {               // Q-U2: U^{n+1} = U^n + dt R(U^n), written to the other buffer
      if ((rc = enqueue_stage(g, 3, g->A, g->A, g->B)) != BATL_OK) return rc;
      if ((rc = enqueue_fill(g, g->B, false)) != BATL_OK) return rc;
      std::swap(g->A, g->B);                   // the buffers trade roles; the caller only sees them through this API
      if ((rc = enqueue_tick(g, 1)) != BATL_OK) return rc;
      continue;
    }
    if ((rc = enqueue_stage(g, 1, g->A, g->A, g->B)) != BATL_OK) return rc;   // U* = U^n + dt/2 R(U^n)
    if ((rc = enqueue_fill(g, g->B, false, b_holds_primitives(g))) != BATL_OK) return rc;
    if ((rc = enqueue_stage(g, 2, g->B, g->A, g->A)) != BATL_OK) return rc;   // U^{n+1} = U^n + dt R(U*)
    if ((rc = enqueue_fill(g, g->A, false)) != BATL_OK) return rc;
    if ((rc = enqueue_tick(g, 1)) != BATL_OK) return rc;                       // t += dt; dt <- min dt_c
  }
  return BATL_OK;
}

int mhd_step(batl_grid* g, int32_t n_steps, double* h_t, double* h_dt_last) {
  int rc = mhd_step_async(g, n_steps);
  if (rc != BATL_OK) return rc;
  DevScalars sc;
  CU(cudaMemcpyAsync(&sc, g->d_scalars(), sizeof(sc), cudaMemcpyDeviceToHost, g->stream));
  CU(cudaStreamSynchronize(g->stream));
  if (g->timers) spans_collect(g);
  if (h_t) *h_t = sc.t;
  if (h_dt_last) *h_dt_last = sc.dt_last;
  if (sc.warn) CU(cudaMemsetAsync(&g->d_scalars()->warn, 0, sizeof(int), g->stream));
  return sc.warn;
}

int batl_get_state(const batl_grid* g, double* h_U, int32_t with_ghost) {
  if (!g || !h_U) return fail(BATL_EINVAL, "null argument");
  if (!g->bound) return fail(BATL_ENOTBOUND, "batl_bind has not been called");
  if (with_ghost == 1 && g->sharded())
    return fail(BATL_EINVAL, "sharded grid: only the own segment is current; use with_ghost = 0 or 2");
  if (with_ghost) {
    if (!g->ghost_full && with_ghost != 2) {          // edge / corner ghosts are only filled on request on the push path
      batl_grid* gm = const_cast<batl_grid*>(g);
      const int rc = enqueue_fill(gm, gm->A, true);
      if (rc != BATL_OK) return rc;
      gm->ghost_full = true;
    }
    CU(cudaMemcpyAsync(h_U, g->A, (size_t)g->h.n_blocks() * BLOCK_BYTES, cudaMemcpyDeviceToHost, g->stream));
  } else {
    CU(launch_gather_phys(g->A, g->B, g->h.n_blocks(), g->stream));
    const_cast<batl_grid*>(g)->launches++;
    CU(cudaMemcpyAsync(h_U, g->B, (size_t)g->h.n_blocks() * NV * NPHYS * sizeof(double), cudaMemcpyDeviceToHost, g->stream));
  }
  CU(cudaStreamSynchronize(g->stream));
  return BATL_OK;
}

int batl_get_dt_local(const batl_grid* g, double* h_dt) {
  if (!g || !h_dt) return fail(BATL_EINVAL, "null argument");
  if (!g->bound) return fail(BATL_ENOTBOUND, "batl_bind has not been called");
  if (g->h.cfg.dt_mode != BATL_DT_LOCAL) return fail(BATL_EINVAL, "dt_mode is not local");
  CU(cudaMemcpyAsync(h_dt, g->d_dtl(), (size_t)g->h.n_blocks() * NPHYS * sizeof(double), cudaMemcpyDeviceToHost, g->stream));
  CU(cudaStreamSynchronize(g->stream));
  return BATL_OK;
}

int batl_set_kernel_variant(batl_grid* g, int32_t variant) {
  if (!g || variant < 0 || variant > 1) return fail(BATL_EINVAL, "bad argument");
  g->variant = variant;
  return BATL_OK;
}

int batl_phase_timers(batl_grid* g, int32_t enable, double* ms_stage, double* ms_ghost, double* ms_other) {
  if (!g) return fail(BATL_EINVAL, "null argument");
  if (g->bound && !g->spans.empty()) { cudaStreamSynchronize(g->stream); spans_collect(g); }
  if (ms_stage) *ms_stage = g->ms_stage;
  if (ms_ghost) *ms_ghost = g->ms_ghost;
  if (ms_other) *ms_other = g->ms_other;
  g->ms_stage = g->ms_ghost = g->ms_other = 0.0;
  g->timers = enable != 0;
  return BATL_OK;
}

int batl_launch_count(const batl_grid* g, int64_t* n) {
  if (!g || !n) return fail(BATL_EINVAL, "null argument");
  *n = g->launches;
  return BATL_OK;
}

int batl_kernel_counts(const batl_grid* g, int64_t* out) {
  if (!g || !out) return fail(BATL_EINVAL, "null argument");
  out[0] = g->n_fused; out[1] = g->n_general; out[2] = g->n_general_fallback;
  out[3] = g->n_fill; out[4] = g->n_fill_blocks; out[5] = (int64_t)g->h.list_fill.size();
  return BATL_OK;
}

}  // extern "C"
