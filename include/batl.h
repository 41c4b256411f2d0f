/* ============================================================================
 * batl.h -- C ABI of the B200-native block-adaptive ideal-MHD step.
 *
 * The hot path of arXiv 2501.06717 ("BATSRUS GPU"), single GPU: one explicit
 * two-stage ideal-MHD time step (fp64) on a block-adaptive Cartesian grid of
 * 8^3-cell blocks with 2 ghost layers.  Citations "L<n>" are line numbers of
 * the paper text; "Q-*" are the readings listed in DESIGN.md for
 * the places where the paper is silent.
 *
 *   state array    : State_VGB(nV, -1:nI+2, -1:nJ+2, -1:nK+2, nB)      L33, L62, L113-117
 *   grid           : root blocks + 2:1 refinement (8 children), tree    L27, L185
 *   ghost fill     : same-level copy, restriction, prolongation, BCs    L64, L115, L128, L146
 *   solver loop    : face value -> face flux -> source -> update        Alg. 1 L29-64, Alg. 2 L76
 *   equations      : ideal MHD, 8-wave source, mu0 = 1                  eqs (1)-(5) L170-183
 *   local exchange : "local message passing" inside one GPU            Alg. 4
 *   index maps     : built on the host once per grid ("IsCounted")      L154-156
 *   data residency : state lives on the GPU, host copy on request       L72, L84
 *
 * Fixed at compile time (L113: block size and nG are fixed before compilation):
 *   nI = nJ = nK = 8, nG = 2, nV = 8, fp64.
 * Variable order (conserved, as stored): 0 rho, 1-3 rho*u, 4-6 B1, 7 e
 *   e = p/(gamma-1) + rho u^2/2 + B1^2/2   (eq. 5; B1 = B - B0 when the
 *   B0 split is on, otherwise B1 = B).
 *
 * Conventions
 *   - every call returns 0 on success, a negative batl_status on error (the
 *     thread-local string of batl_last_error() says why); mhd_step may return
 *     a positive warning bitmask (BATL_WARN_*).
 *   - no exceptions cross the ABI, no global state except the error string;
 *     every batl_grid is independent (replicas on several GPUs = several grids).
 *   - "h_" pointers are HOST memory, "d_" pointers are DEVICE memory.  The
 *     library never allocates or frees device memory: the caller owns the
 *     state buffers, the scratch buffer and the stream (PyTorch tensors / a
 *     PyTorch stream in the Python binding) and must keep them alive while
 *     the grid is bound to them.
 *   - block order seen by the caller is the library's Morton order (Q-O1):
 *     sort leaves by root index Ix + nx (Iy + ny Iz), then by the child digits
 *     ox + 2 oy + 4 oz from the top level down.
 *   - geometry of block (level, I, J, K):
 *       D_a   = (max_a - min_a) / (8 n_root_a) * 2^-level
 *       x_a   = min_a + (8 I_a + i + 1/2) D_a            cell centre, i = 0..7
 *   - device layout of a state buffer: [block][var][k][j][i] with 12^3 doubles
 *     per variable (storage index s = i + 2; ghosts i in {-2,-1,8,9}),
 *     110,592 bytes per block.
 * ========================================================================== */
#ifndef BATL_H_
#define BATL_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum batl_status {
  BATL_OK = 0,
  BATL_EINVAL = -1,   /* invalid argument                                       */
  BATL_ENOMEM = -2,   /* host allocation failed / caller buffer too small       */
  BATL_ECUDA = -3,    /* a CUDA call failed (no device, launch error, ...)      */
  BATL_EGRID = -4,    /* periodic faces not paired, regions inconsistent        */
  BATL_ENOTBOUND = -5 /* batl_bind has not been called                          */
};

enum { BATL_WARN_NONFINITE = 1, /* non-finite rho or p seen on a stage's input    */
       BATL_WARN_NEGATIVE = 2   /* rho <= 0 or p <= 0 seen on a stage's input     */ };

enum { BATL_BC_PERIODIC = 0, BATL_BC_FLOAT = 1, BATL_BC_FIXED = 2 };
enum { BATL_SHAPE_ALL = 0, BATL_SHAPE_BOX = 1, BATL_SHAPE_SPHERE = 2 };
enum { BATL_DT_GLOBAL = 0, BATL_DT_LOCAL = 1, BATL_DT_FIXED = 2 };

/* ghost-list formats of batl_get_ghost_list */
enum { BATL_LIST_MESSAGES = 0, /* batl_ghost_msg records (region form of the lists)  */
       BATL_LIST_EXPANDED = 1, /* int32[9] per ghost cell, canonical form (below),
                                * expanded from the message records                 */
       BATL_LIST_PLAN = 2,     /* the same int32[9] tuples, decoded from the per-cell
                                * plan the ghost-fill kernel reads                  */
       BATL_LIST_PLAN_PATTERNS = 3, /* uint32[n][1216]: the distinct per-cell plan
                                * patterns (blocks with equal surroundings share one) */
       BATL_LIST_PLAN_IDS = 4, /* int32[nB]: the pattern of each block               */
       BATL_LIST_FC_SLOTS = 5, /* int32[nB][6]: flux-correction slot of every block face
                                * at a resolution change, -1 otherwise (Q-G6b)       */
       BATL_LIST_FC_RECORDS = 6 /* int32[n][8]: per face that borders finer blocks: block,
                                * face, own slot, slots of the four fine faces (lower
                                * tangential axis fastest), 0                        */ };
/* kinds of a ghost message / of an expanded tuple (L128: three message types;
 * boundary conditions L64) */
enum { BATL_MSG_COPY = 0, BATL_MSG_RESTRICT = 1, BATL_MSG_PROLONG = 2, BATL_MSG_FIXED = 3 };

typedef struct batl_grid batl_grid; /* opaque; created and destroyed only by the library */

/* Refinement region: every leaf whose OPEN block box intersects the shape is
 * refined until it reaches `level` (L185: "one octant refined"; L391).
 *   shape BOX    : p = {lo_x, lo_y, lo_z, hi_x, hi_y, hi_z}
 *   shape SPHERE : p = {c_x, c_y, c_z, radius, -, -}   (min distance box-centre < radius)
 *   shape ALL    : p unused */
typedef struct {
  int32_t shape;
  int32_t level;
  double p[6];
} batl_region;

/* Plain data, copied at batl_init_grid; the caller keeps ownership of `region`. */
typedef struct {
  int32_t n_root[3];            /* root blocks per axis (L185)                           */
  double xyz_min[3], xyz_max[3];
  int32_t bc[6];                /* -x,+x,-y,+y,-z,+z: BATL_BC_*; periodic must pair (L64, L343) */
  double bc_prim[6][8];         /* primitive (rho, u, B1, p) of BATL_BC_FIXED faces      */
  int32_t n_region;
  const batl_region* region;    /* host pointer, n_region entries (may be NULL if 0)     */
  int32_t max_level;            /* no leaf is refined by a region beyond this level      */
  double gamma;                 /* ratio of specific heats (eq. 5)                       */
  double cfl;                   /* CFL number (L343: 0.8)                                */
  double limiter_beta;          /* MC(beta) limiter parameter, 2.0 = monotonised central */
  int32_t dt_mode;              /* BATL_DT_*: global (lagged, Q-T2), local (L389), fixed */
  double dt_fixed;
  int32_t use_divb_source;      /* 8-wave source terms of eqs (2)-(4) (L170-183)         */
  int32_t use_b0;               /* 1: B = B0 + B1 with B0 the analytic dipole dipole_m at
                                 * the origin; 2: uniform B0 = dipole_m (test aid)       */
  double dipole_m[3];
  int32_t use_body;             /* spherical inner boundary at the origin (L391)         */
  double r_body, rho_body, p_body; /* p_body <= 0: pressure floats at the body           */
  int32_t n_stage;              /* 2: two-stage scheme (Q-U1, the default when 0);
                                 * 1: one stage, first order in time (L391-397):
                                 *    U^{n+1} = U^n + dt R(U^n), ghost fill              */
  int32_t n_order;              /* 2: limited linear face states (default when 0);
                                 * 1: piecewise-constant face states (L86 "nOrder")      */
  int32_t flux_type;            /* 0: Rusanov (Q-F1); 1: HLL-type two-wave flux, the
                                 * reading Q-F4 of the paper's "Linde flux" (L343)       */
  int32_t prolong_order;        /* resolution changes (L128 names the operations and gives no
                                 * formula).  1 (default when 0): a fine
                                 * ghost cell takes the value of the coarse cell that contains
                                 * it (Q-G4).  2: it takes the coarse cell's MC(beta)-limited
                                 * linear profile at its own centre, U_C +- s_d/4 per axis
                                 * (Q-G4b); the fill then runs in two passes (copy, restriction
                                 * and boundary states first, prolongation second)          */
  int32_t flux_correction;      /* 1: the flux through a face cell that borders FINER blocks is
                                 * replaced by the mean of the four fine face fluxes before the
                                 * update, in every stage (Q-G6b): the scheme then conserves on
                                 * AMR grids ("nearly conservative form", L168).  0: none (Q-G6) */
} batl_config;

/* One ghost region of one destination block, filled from ONE source block (or
 * from a fixed boundary state).  Destination cells: lo[a] .. lo[a]+n[a]-1 along
 * axis a (cell indices, ghosts are -2,-1,8,9).  Source cell along axis a for a
 * destination cell c:   s = (mul[a]*c + off[a]) >> shift[a]
 *   COPY     mul 1, shift 0   (mul 0: coordinate clamped at a float boundary)
 *   PROLONG  shift 1          (first order: value of the containing coarse cell, Q-G4)
 *   RESTRICT mul 2            (s = lowest of the 2x2x2 fine cells; mean in the fixed
 *                              pairwise order x, then y, then z, Q-G3)
 *   FIXED    src = -2-face    (value = conserved form of bc_prim[face]) */
typedef struct {
  int32_t dst, src;
  int8_t kind, dir;             /* dir = (di+1)+3(dj+1)+9(dk+1) of the region, 13 never  */
  int8_t lo[3], n[3];
  int8_t mul[3], off[3], shift[3];
  int8_t pad[3];
} batl_ghost_msg;               /* 28 bytes */

/* Build the block tree, the Morton order, the neighbour table and the ghost
 * messages on the HOST (L27, L128, L154-156).  Touches no CUDA API, so it runs
 * on a machine without a GPU.  *out must be released with batl_free_grid. */
int batl_init_grid(const batl_config* cfg, batl_grid** out);
void batl_free_grid(batl_grid* g);

int batl_n_blocks(const batl_grid* g, int32_t* n_blocks);

/* Sizes of the caller-owned device buffers: each of the two state buffers
 * (state_bytes = n_blocks * 110592 + 256: the tiles start 16 bytes into the buffer,
 * DESIGN.md section 5) and the scratch buffer (tables, per-cell
 * local time steps, scalars). */
int batl_buffer_bytes(const batl_grid* g, size_t* state_bytes, size_t* scratch_bytes);

/* Attach the device buffers and the stream (a cudaStream_t cast to void*, NULL =
 * legacy default stream) and upload the tables into d_scratch.  d_* must be
 * 256-byte aligned.  Everything the library later does is enqueued on this
 * stream.  Fails with BATL_ECUDA if there is no usable device. */
int batl_bind(batl_grid* g, void* d_stateA, void* d_stateB, void* d_scratch, void* cuda_stream);

/* Upload the conserved state of the physical cells, h_U[nB][8][8][8][8] =
 * [block][var][k][j][i] (host), fill all ghost cells, reset t = 0 and the
 * lagged time step.  batl_set_state_device takes the same array from device
 * memory (no host copy; used when the data is already resident in HBM).
 * Stream ordering: both copies are enqueued on the bound stream.  d_U must be complete
 * with respect to that stream when batl_set_state_device is called (the caller orders
 * its producer stream before the bound one, e.g. with an event; the Python binding does)
 * and must stay allocated until the stream has passed the copy. */
int batl_set_state(batl_grid* g, const double* h_U);
int batl_set_state_device(batl_grid* g, const double* d_U);

/* Advance n_steps steps.  Two-stage scheme (Q-U1):
 *   U* = U^n + dt/2 R(U^n); ghost fill; U^{n+1} = U^n + dt R(U*); ghost fill; t += dt
 * One-stage scheme (n_stage = 1, Q-U2): U^{n+1} = U^n + dt R(U^n); ghost fill; t += dt
 * All launches go to the bound stream without host synchronisation; the call
 * then waits for the stream and reads back t, the last dt and the warning
 * bits (h_t / h_dt_last may be NULL).  Returns <0 on error, else BATL_WARN_* bits.
 * mhd_step_async enqueues the same work and returns without waiting. */
int mhd_step(batl_grid* g, int32_t n_steps, double* h_t, double* h_dt_last);
int mhd_step_async(batl_grid* g, int32_t n_steps);

/* Ghost fill of the current state alone (steps a1-a4): every ghost cell of every block
 * (faces, edges, corners; L146), enqueued on the stream.  Inside mhd_step the product
 * path does not run this pass for same-level faces: the stage kernels write the two outer
 * cell layers of a block into the face-ghost slots of its same-level neighbours (the
 * scheme reads no edge or corner ghost), and only blocks with a face at a resolution
 * change or a non-periodic boundary are filled by the plan-driven kernel.  Edge and
 * corner ghosts of the other blocks are therefore brought up to date only by this call
 * or by batl_get_state(with_ghost = 1), which runs it first when needed. */
int batl_fill_ghosts(batl_grid* g);

/* Download the state: with_ghost = 0 -> h_U[nB][8][8][8][8], 1 -> [nB][8][12][12][12]
 * (all 26 ghost regions current, see batl_fill_ghosts), 2 -> the same array as it sits in
 * device memory, without the fill on request (what the next stage kernel would read: the
 * parity tests check the pushed face ghosts with it).  Synchronises the stream.
 * batl_set_state / batl_set_state_device / batl_get_state(with_ghost = 0) use state
 * buffer B as staging area: its contents are undefined afterwards (it only ever holds
 * the intermediate state U* inside a step).  batl_get_dt_local: h_dt[nB][8][8][8] (dt_mode local). */
int batl_get_state(const batl_grid* g, double* h_U, int32_t with_ghost);
int batl_get_dt_local(const batl_grid* g, double* h_dt);

/* Introspection (host data, no CUDA): what "bit-exact" parity is judged on.
 *   lvl_ijk[nB][4]   = (level, I, J, K) in block order
 *   nbr[nB][27][4]   block ids per direction dir = (di+1)+3(dj+1)+9(dk+1) (13 = self):
 *                    one id for a same-level or coarser neighbour; for finer ones
 *                    4 (face) / 2 (edge) / 1 (corner) ids, lower tangential axis
 *                    fastest; -1 padding
 *   dlev[nB][27]     0 same level, +1 neighbour coarser, -1 finer, -100 outside a
 *                    non-periodic boundary
 *   ghost list       kind MESSAGES: batl_ghost_msg[n]; kind EXPANDED: int32[n][9] =
 *                    (dst_block, k, j, i, kind, src_block, k', j', i') per ghost cell,
 *                    sorted lexicographically (restriction: lowest fine cell of the 8;
 *                    fixed BC: src_block = -2-face, k'=j'=i'=0).
 *                    Call with out = NULL to get the count in *n. */
int batl_get_blocks(const batl_grid* g, int32_t* lvl_ijk);
int batl_get_neighbors(const batl_grid* g, int32_t* nbr, int8_t* dlev);
int batl_get_ghost_list(const batl_grid* g, int32_t kind, void* out, size_t* n);

/* Kernel selection for measurements and parity tests: 0 = fused shared-memory
 * stage kernel where it applies (default), 1 = general reference kernel everywhere. */
int batl_set_kernel_variant(batl_grid* g, int32_t variant);

/* Opt-in per-phase timers (the paper's "Process Buffer" / "Update State" split,
 * Table 3): accumulated CUDA-event milliseconds of the stage kernels,
 * the ghost fills and the dt bookkeeping since the last reset.  enable = 1 makes
 * mhd_step record events around every launch. */
int batl_phase_timers(batl_grid* g, int32_t enable, double* ms_stage, double* ms_ghost, double* ms_other);

/* Number of kernel launches the library has enqueued since the grid was bound. */
int batl_launch_count(const batl_grid* g, int64_t* n);

/* Which kernels mhd_step has used since the grid was bound, out[6] (host):
 *   [0] launches of the fused stage kernel
 *   [1] launches of the general stage kernel (blocks with body cells; reference path)
 *   [2] of [1], launches that took EVERY block although the fused kernel was asked for
 *       (kernel variant 0) because it has no instantiation for the configuration --
 *       about three times slower; 0 on every BASELINE.json config
 *   [3] ghost-fill launches, [4] destination blocks they filled in total
 *   [5] number of blocks on the fill list (blocks with a face at a resolution change
 *       or a non-periodic boundary; all other face ghosts are written by the stage
 *       kernels themselves) */
int batl_kernel_counts(const batl_grid* g, int64_t* out);

/* ---- Sharding over the GPUs of one node ("contiguous blocks per
 * rank", section 4.4, Alg. 4) --------------------------------------------------------------
 * One process per GPU, every process builds the SAME grid (the tree lives on every rank, L27) and owns
 * a contiguous segment of the Morton-ordered blocks.  There is no message buffer: the state buffers of
 * all ranks are mapped into every process (CUDA IPC over NVLink; the caller does the mapping and passes
 * the pointers), the stage kernel writes the two outer cell layers of its blocks straight into the
 * face-ghost slots of neighbours that live on another GPU, and the fill kernel reads source blocks
 * from the owner's buffer.  The library enqueues the parts of a step; BETWEEN them the caller
 * synchronises the ranks on the bound stream (a barrier after each stage) and, for dt_mode global,
 * all-reduces (min) the 8 bytes at scratch + *dt_next_offset, which hold the bit pattern of a positive
 * double (its order as an unsigned integer is the order of the doubles).  Sequence of one step:
 *     [first step after batl_set_state, dt_mode global: DT0, all-reduce, TICK_START]
 *     STAGE1, barrier, FILL_B, STAGE2, barrier, FILL_A, all-reduce (doubles as the barrier), TICK_END
 * batl_set_state takes the whole initial state on every rank; afterwards a rank's buffers are current
 * for its own blocks and their face ghosts only, and batl_get_state(with_ghost = 0) returns the whole
 * array with only the own segment valid.  One-stage scheme (n_stage = 1): STAGE1 is the single stage,
 * then barrier, FILL_B, all-reduce, TICK_END (which trades the buffers on every rank); STAGE2 and FILL_A
 * enqueue nothing.  Supported: both schemes, every dt_mode, first-order prolongation, no flux correction
 * (these two need a further exchange); kernel variant 0.
 * batl_set_partition must precede batl_bind; world = 1 restores the unsharded grid. */
enum { BATL_PART_DT0 = 0, BATL_PART_TICK_START = 1, BATL_PART_STAGE1 = 2, BATL_PART_FILL_B = 3,
       BATL_PART_STAGE2 = 4, BATL_PART_FILL_A = 5, BATL_PART_TICK_END = 6 };
int batl_set_partition(batl_grid* g, int32_t world, int32_t rank);
/* first_block[world + 1]: rank r owns blocks first_block[r] .. first_block[r + 1] - 1 */
int batl_get_partition(const batl_grid* g, int32_t* first_block);
/* d_stateA[world], d_stateB[world] (host arrays of device pointers): the state buffers of every rank as
 * mapped into THIS process; entry `rank` must be the buffers given to batl_bind. */
int batl_bind_peers(batl_grid* g, void* const* d_stateA, void* const* d_stateB);
int batl_step_part(batl_grid* g, int32_t part);
int batl_scalar_offsets(const batl_grid* g, size_t* dt_next_offset);

const char* batl_last_error(void); /* thread-local, library-owned string */

/* ---- Entry point that allocates nothing and needs no caller-owned scratch buffer -------------------
 * For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid it) and therefore cannot size and hand over the scratch buffer of batl_bind.
 *
 * mhd_stable_dt_static: the stable (CFL) time step of a tiled state, the "calculate time step" of the
 * solver loop (Alg. 1 L29-64; CFL number L343; step a9, readings Q-T1 / Q-T2 of DESIGN.md):
 *     dt = min over the physical cells c of all blocks of  cfl / sum_d max(c_d(c-1/2), c_d(c+1/2)) / D_d
 * with c_d the wave speed of the face flux (Rusanov: max |u_n| + c_fast of the two face states; flux_type
 * 1: the HLL-type bound, Q-F4) at the limited face states (n_order 2, MC limiter with limiter_beta) or
 * the cell values (n_order 1).  It is the same kernel pass that gives a bound grid the dt of its first
 * step (stage 0 of the general stage kernel), with the working data that pass keeps in the scratch
 * buffer of batl_bind -- the per-block geometry table, the running minimum, the warning bits -- held
 * in a file-scope device array of the library instead.
 *   d_tiles      device, [n_blocks][8][12][12][12] doubles: conserved variables in the device layout
 *                of a state buffer (see top of this file), ghost cells of all six faces current.  For
 *                a bound grid this is stateA + 16 bytes after batl_set_state / mhd_step.  Read only.
 *   d_cell_size  device, [n_blocks][3] doubles: cell size (D_x, D_y, D_z) of each block.  Read only.
 *   n_blocks     1 .. BATL_STATIC_MAX_BLOCKS; more is refused with BATL_ENOMEM and a message that
 *                states the limit (nothing is enqueued).
 *   gamma, cfl, limiter_beta, n_order (0 = 2), flux_type, use_divb_source: as in batl_config.  B0
 *                split and body cells are not offered (they need the grid's tables).
 *   d_dt         device, 1 double: receives dt (+inf if no cell has a positive finite limit).
 *   d_warn       device, 1 int32, or NULL: receives the BATL_WARN_* bits of the input state.
 *   cuda_stream  the three kernels of the call are enqueued on it; the call does not wait.
 * Ownership: the caller owns every pointer and keeps them alive until the stream has passed the call.
 * The library's static array (BATL_STATIC_MAX_BLOCKS * 88 + 256 = 360,704 bytes of device memory on
 * every GPU that loads the library, until the process exits) is shared by ALL calls and keeps the last
 * call's contents; each call rewrites what it reads before reading it, so calls on one stream (or
 * otherwise ordered on the GPU) are independent, while calls that OVERLAP on the GPU race on it and
 * give undefined results.  The call makes no cudaMalloc / cudaFree and no other allocating call; the
 * first call on a device looks up the array's address and sets the kernel's shared-memory attribute.
 * Errors: negative batl_status, text in batl_static_last_error() (thread-local, library-owned). */
#define BATL_STATIC_MAX_BLOCKS 4096
int mhd_stable_dt_static(const double* d_tiles, const double* d_cell_size, int32_t n_blocks, double gamma,
                         double cfl, double limiter_beta, int32_t n_order, int32_t flux_type,
                         int32_t use_divb_source, double* d_dt, int32_t* d_warn, void* cuda_stream);
const char* batl_static_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* BATL_H_ */
