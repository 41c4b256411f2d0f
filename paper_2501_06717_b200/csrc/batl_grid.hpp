// Host side of the library: block tree, Morton order, neighbour table and ghost
// messages (steps a0 of the hot path; the index
// maps are built serially on the host once per grid and reused until it changes).
// Pure C++; nothing here touches CUDA.
#pragma once
#include <cstdint>
#include <string>
#include <unordered_map>
#include <vector>

#include "batl.h"

namespace batl {

constexpr int NI = 8;                 // cells per block and axis (L391)
constexpr int NG = 2;                 // ghost layers (L113)
constexpr int NS = NI + 2 * NG;       // stored cells per axis
constexpr int NV = 8;                 // variables
constexpr int NCELL = NS * NS * NS;   // 1728 stored cells per block and variable
constexpr int NPHYS = NI * NI * NI;   // 512
constexpr size_t BLOCK_DOUBLES = (size_t)NV * NCELL;
constexpr size_t BLOCK_BYTES = BLOCK_DOUBLES * sizeof(double);   // 110,592

struct Leaf {
  int32_t level;
  int32_t I[3];
};

// per-block data the kernels read (uploaded as is)
struct BlockGeom {
  double x0[3];      // coordinate of the low corner of cell 0:  min_a + 8 I_a D_a
  double D[3];       // cell size D_a
  double invD[3];    // 1 / D_a, scaled from the root value by an exact power of two
  int32_t level;
  int32_t flags;     // bit 0: block contains body cells among its 12^3 stored cells
  int32_t mask_slot; // index into the body-mask table, -1 if none
  int32_t pad;
};
constexpr int BODY_MASK_WORDS = NCELL / 32;   // 54 uint32 per flagged block

// Per-cell ghost plan (what ghost_fill_kernel reads): the messages of a block expanded
// to one 32-bit entry per ghost cell, in storage order of the destination cell.
//   bits  0-10  destination cell (storage offset in a 12^3 variable)
//   bits 11-21  source cell (storage offset; RESTRICT: lowest of the 8 fine cells;
//               FIXED: boundary face 0..5)
//   bits 22-27  slot of the source block in the block's source list
//   bits 28-31  PLAN_COPY (copy, first-order prolongation, float boundary) / PLAN_RESTRICT / PLAN_FIXED /
//               PLAN_PROLONG2 | px | py << 1 | pz << 2 (second-order prolongation, Q-G4b: source = the
//               coarse cell, p = 1 if the fine cell is the high child of it along that axis)
// Entries hold no block id, so blocks with the same surroundings share one pattern
// (a uniform periodic grid has exactly one); block ids sit in plan_src[b][slot].
constexpr int NGHOST = NCELL - NPHYS;         // 1216 ghost cells per block
constexpr int PLAN_SLOTS = 64;                // >= 6*4 + 12*2 + 8 finer neighbours + the block itself
enum { PLAN_COPY = 0, PLAN_RESTRICT = 1, PLAN_FIXED = 2, PLAN_PROLONG2 = 8 };
constexpr int32_t PUSH_BY_COARSER = -(1 << 30);

struct HostGrid {
  batl_config cfg;
  std::vector<batl_region> regions;
  std::vector<Leaf> leaf;                         // Morton order (Q-O1)
  std::unordered_map<uint64_t, int32_t> index;    // (level, I, J, K) -> block id
  std::vector<int32_t> nbr;                       // [nB][27][4]
  std::vector<int8_t> dlev;                       // [nB][27]
  std::vector<batl_ghost_msg> msg;                // grouped by destination block
  std::vector<int32_t> msg_start;                 // [nB + 1]
  std::vector<uint32_t> plan;                     // [n_pattern][NGHOST]
  std::vector<int32_t> plan_id;                   // [nB] pattern of each block
  std::vector<int32_t> plan_src;                  // [nB][PLAN_SLOTS] source block ids, -1 padding
  std::vector<BlockGeom> geom;                    // [nB]
  std::vector<int32_t> list_plain, list_body;     // blocks without / with body cells among their stored cells
  // Ghost cells without a stored-ghost pass: the stage kernels write the two
  // outer cell layers of a block straight into the face-ghost slots of its same-level face
  // neighbours.  push_nbr[b][f], f = -x,+x,-y,+y,-z,+z: that neighbour's id, -1 if the face is at a
  // resolution change or a non-periodic boundary.  list_fill: the blocks with at least one such
  // face; only they still need the plan-driven fill after a stage.
  // Values < 0 of push_nbr: -1 = nobody writes these face ghosts (boundary face; any resolution change under
  // second-order prolongation): the fill pass does; -2 - n = FINER neighbours, ids in push_fine[n][0..3] (lower
  // tangential axis fastest): the stage kernel pushes first-order prolonged values into THEIR ghosts, and the
  // fill pass restricts into ours; PUSH_BY_COARSER = the coarser neighbour pushes into ours: nothing to fill.
  std::vector<int32_t> push_nbr;                  // [nB][6]
  std::vector<int32_t> push_fine;                 // [n][4]
  std::vector<int32_t> list_fill;
  std::vector<int32_t> list_prolong;              // blocks with second-order prolonged ghost cells (Q-G4b)
  // Flux correction (Q-G6b).  fc_slot[b][f]: slot of the face-flux buffer ([slot][var][t_hi][t_lo], the
  // tangential axes in ascending order) for a face at a resolution change, -1 otherwise.  fc_list: one
  // record of 8 int32 per face that borders finer blocks: block, face, own slot, the slots of the four
  // fine faces (lower tangential axis fastest), 0.
  std::vector<int32_t> fc_slot;                   // [nB][6]
  std::vector<int32_t> fc_list;                   // [n][8], sorted by block
  std::vector<int32_t> fc_group;                  // [n_blocks_with_records][2]: first record, number of records
                                                  // (a cell at an edge or corner is corrected through 2 or 3
                                                  // faces: one CTA takes all faces of a block, in order)
  int32_t n_fc_slots = 0;
  std::vector<uint32_t> body_mask;                // [n_mask][54], bit s = stored cell s is a body cell
  double bc_cons[6][NV];                          // conserved form of bc_prim (eq. 5)
  int max_level_present = 0;

  int n_blocks() const { return (int)leaf.size(); }
};

// Builds everything above.  Returns BATL_OK or a negative status with `err` set.
int build_grid(const batl_config& cfg, HostGrid& g, std::string& err);

// expanded canonical ghost list: (dst, k, j, i, kind, src, k', j', i') per ghost cell
void expand_ghost_list(const HostGrid& g, std::vector<int32_t>& out);
// the same tuples decoded from the per-cell plan (plan, plan_id, plan_src)
void expand_plan_list(const HostGrid& g, std::vector<int32_t>& out);

}  // namespace batl
