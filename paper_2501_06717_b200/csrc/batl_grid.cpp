// Host builder: block tree -> Morton order -> neighbour table -> ghost messages.
// PAPER.md L27 (tree, 2:1 refinement, 8 children), L128 (three message types and
// their index ranges), L154-156 (maps built once on the host, "IsCounted").
// The readings Q-O1..Q-O3, Q-G1..Q-G5 are stated in DESIGN.md.
#include "batl_grid.hpp"

#include <algorithm>
#include <cmath>
#include <string>
#include <unordered_map>
#include <unordered_set>

namespace batl {
namespace {

inline uint64_t pack(int level, int i, int j, int k) {
  return ((uint64_t)level << 57) | ((uint64_t)(uint32_t)i << 38) | ((uint64_t)(uint32_t)j << 19) |
         (uint64_t)(uint32_t)k;
}
inline Leaf unpack(uint64_t key) {
  Leaf L;
  L.level = (int)(key >> 57);
  L.I[0] = (int)((key >> 38) & 0x7FFFF);
  L.I[1] = (int)((key >> 19) & 0x7FFFF);
  L.I[2] = (int)(key & 0x7FFFF);
  return L;
}

// geometry contract of batl.h
inline double block_edge(const batl_config& c, int a, int level) {
  return std::ldexp((c.xyz_max[a] - c.xyz_min[a]) / c.n_root[a], -level);
}

bool box_hits_region(const batl_config& c, const Leaf& L, const batl_region& r) {
  if (r.shape == BATL_SHAPE_ALL) return true;
  double lo[3], hi[3];
  for (int a = 0; a < 3; ++a) {
    const double s = block_edge(c, a, L.level);
    lo[a] = c.xyz_min[a] + L.I[a] * s;
    hi[a] = c.xyz_min[a] + (L.I[a] + 1) * s;
  }
  if (r.shape == BATL_SHAPE_BOX) {
    for (int a = 0; a < 3; ++a)
      if (!(lo[a] < r.p[3 + a] && hi[a] > r.p[a])) return false;
    return true;
  }
  double d2 = 0.0;   // sphere: distance from the centre to the box
  for (int a = 0; a < 3; ++a) {
    double d = 0.0;
    if (r.p[a] < lo[a]) d = lo[a] - r.p[a];
    else if (r.p[a] > hi[a]) d = r.p[a] - hi[a];
    d2 += d * d;
  }
  return d2 < r.p[3] * r.p[3];
}

struct Tree {
  const batl_config& c;
  std::unordered_set<uint64_t> leaves;
  explicit Tree(const batl_config& cfg) : c(cfg) {}

  void split(const Leaf& L) {
    leaves.erase(pack(L.level, L.I[0], L.I[1], L.I[2]));
    for (int o = 0; o < 8; ++o)
      leaves.insert(pack(L.level + 1, 2 * L.I[0] + (o & 1), 2 * L.I[1] + ((o >> 1) & 1), 2 * L.I[2] + (o >> 2)));
  }
  // leaf that contains block position P of `level`; 0 if the position is covered by finer leaves
  bool containing(int level, const int P[3], uint64_t* key) const {
    for (int l = level; l >= 0; --l) {
      const int s = level - l;
      const uint64_t k = pack(l, P[0] >> s, P[1] >> s, P[2] >> s);
      if (leaves.count(k)) { *key = k; return true; }
    }
    return false;
  }
  // neighbour position with periodic wrap; false if outside a non-periodic face
  bool shifted(const Leaf& L, const int d[3], int P[3]) const {
    for (int a = 0; a < 3; ++a) {
      const int N = c.n_root[a] << L.level;
      P[a] = L.I[a] + d[a];
      if (P[a] < 0 || P[a] >= N) {
        if (c.bc[2 * a + (P[a] >= N ? 1 : 0)] != BATL_BC_PERIODIC) return false;
        P[a] = (P[a] + N) % N;
      }
    }
    return true;
  }
};

}  // namespace

int build_grid(const batl_config& cfg, HostGrid& g, std::string& err) {
  // ---------------------------------------------------------------- checks --
  for (int a = 0; a < 3; ++a) {
    if (cfg.n_root[a] < 1 || cfg.n_root[a] > 4096) { err = "n_root out of range"; return BATL_EINVAL; }
    if (!(cfg.xyz_max[a] > cfg.xyz_min[a])) { err = "xyz_max must exceed xyz_min"; return BATL_EINVAL; }
    const int lo = cfg.bc[2 * a], hi = cfg.bc[2 * a + 1];
    if (lo < 0 || lo > 2 || hi < 0 || hi > 2) { err = "unknown boundary type"; return BATL_EINVAL; }
    if ((lo == BATL_BC_PERIODIC) != (hi == BATL_BC_PERIODIC)) { err = "periodic faces must pair"; return BATL_EGRID; }
  }
  if (cfg.max_level < 0 || cfg.max_level > 12) { err = "max_level out of range [0,12]"; return BATL_EINVAL; }
  for (int a = 0; a < 3; ++a)
    if (((int64_t)cfg.n_root[a] << cfg.max_level) >= (1 << 19)) { err = "n_root << max_level must stay below 2^19"; return BATL_EINVAL; }
  if (cfg.n_region < 0 || (cfg.n_region > 0 && !cfg.region)) { err = "region list missing"; return BATL_EINVAL; }
  if (!(cfg.gamma > 1.0)) { err = "gamma must exceed 1"; return BATL_EINVAL; }
  if (!(cfg.cfl > 0.0) || !(cfg.limiter_beta >= 1.0)) { err = "cfl > 0 and limiter_beta >= 1 required"; return BATL_EINVAL; }
  if (cfg.dt_mode < 0 || cfg.dt_mode > 2) { err = "unknown dt_mode"; return BATL_EINVAL; }
  if (cfg.dt_mode == BATL_DT_FIXED && !(cfg.dt_fixed > 0.0)) { err = "dt_fixed must be positive"; return BATL_EINVAL; }
  if (cfg.use_b0 < 0 || cfg.use_b0 > 2) { err = "unknown use_b0"; return BATL_EINVAL; }
  for (int r = 0; r < cfg.n_region; ++r) {
    if (cfg.region[r].shape < 0 || cfg.region[r].shape > 2 || cfg.region[r].level < 0) {
      err = "bad refinement region"; return BATL_EGRID;
    }
  }
  if (cfg.n_stage < 0 || cfg.n_stage > 2 || cfg.n_order < 0 || cfg.n_order > 2) { err = "n_stage and n_order must be 1 or 2 (0 = default 2)"; return BATL_EINVAL; }
  if (cfg.flux_type < 0 || cfg.flux_type > 1) { err = "unknown flux_type"; return BATL_EINVAL; }
  if (cfg.prolong_order < 0 || cfg.prolong_order > 2) { err = "prolong_order must be 1 or 2 (0 = default 1)"; return BATL_EINVAL; }
  if (cfg.flux_correction < 0 || cfg.flux_correction > 1) { err = "flux_correction must be 0 or 1"; return BATL_EINVAL; }
  g.cfg = cfg;
  if (g.cfg.n_stage == 0) g.cfg.n_stage = 2;
  if (g.cfg.n_order == 0) g.cfg.n_order = 2;
  if (g.cfg.prolong_order == 0) g.cfg.prolong_order = 1;
  g.regions.assign(cfg.region, cfg.region + cfg.n_region);
  g.cfg.region = nullptr;

  // -------------------------------------------------- leaves from the regions --
  Tree T(g.cfg);
  for (int k = 0; k < cfg.n_root[2]; ++k)
    for (int j = 0; j < cfg.n_root[1]; ++j)
      for (int i = 0; i < cfg.n_root[0]; ++i) T.leaves.insert(pack(0, i, j, k));

  std::vector<uint64_t> work(T.leaves.begin(), T.leaves.end());
  while (!work.empty()) {                       // each new child is examined once
    const uint64_t key = work.back();
    work.pop_back();
    const Leaf L = unpack(key);
    if (L.level >= cfg.max_level) continue;
    bool hit = false;
    for (const batl_region& r : g.regions)
      if (L.level < r.level && box_hits_region(g.cfg, L, r)) { hit = true; break; }
    if (!hit) continue;
    T.split(L);
    for (int o = 0; o < 8; ++o)
      work.push_back(pack(L.level + 1, 2 * L.I[0] + (o & 1), 2 * L.I[1] + ((o >> 1) & 1), 2 * L.I[2] + (o >> 2)));
  }

  // ------------------------------ 2:1 nesting over faces, edges, corners (Q-O2) --
  // A leaf is split if any of the 26 same-size neighbour positions of a leaf two or
  // more levels finer falls inside it.  The closure is unique, so the order of
  // splitting does not matter.
  for (;;) {
    std::unordered_set<uint64_t> marked;
    for (const uint64_t key : T.leaves) {
      const Leaf L = unpack(key);
      if (L.level < 2) continue;
      for (int q = 0; q < 27; ++q) {
        if (q == 13) continue;
        const int d[3] = {q % 3 - 1, (q / 3) % 3 - 1, q / 9 - 1};
        int P[3];
        if (!T.shifted(L, d, P)) continue;
        uint64_t nk;
        if (T.containing(L.level, P, &nk) && (int)(nk >> 57) < L.level - 1) marked.insert(nk);
      }
    }
    if (marked.empty()) break;
    for (const uint64_t k : marked) T.split(unpack(k));
  }

  // ------------------------------------------------------ Morton order (Q-O1) --
  int lmax = 0;
  for (const uint64_t k : T.leaves) lmax = std::max(lmax, (int)(k >> 57));
  g.max_level_present = lmax;
  struct Keyed { uint64_t root, digits; Leaf L; };
  std::vector<Keyed> order;
  order.reserve(T.leaves.size());
  for (const uint64_t k : T.leaves) {
    Keyed e;
    e.L = unpack(k);
    const int lev = e.L.level;
    const uint64_t r0 = e.L.I[0] >> lev, r1 = e.L.I[1] >> lev, r2 = e.L.I[2] >> lev;
    e.root = r0 + (uint64_t)cfg.n_root[0] * (r1 + (uint64_t)cfg.n_root[1] * r2);
    e.digits = 0;
    for (int l = 1; l <= lev; ++l) {            // child digits from the top level down
      const int sh = lev - l;
      const uint64_t dgt = ((e.L.I[0] >> sh) & 1) + 2 * ((e.L.I[1] >> sh) & 1) + 4 * ((e.L.I[2] >> sh) & 1);
      e.digits |= dgt << (3 * (lmax - l));      // left aligned: leaves are never prefixes of one another
    }
    order.push_back(e);
  }
  std::sort(order.begin(), order.end(), [](const Keyed& a, const Keyed& b) {
    return a.root != b.root ? a.root < b.root : a.digits < b.digits;
  });
  const int nB = (int)order.size();
  g.leaf.resize(nB);
  g.index.clear();
  g.index.reserve((size_t)nB * 2);
  for (int b = 0; b < nB; ++b) {
    g.leaf[b] = order[b].L;
    g.index[pack(order[b].L.level, order[b].L.I[0], order[b].L.I[1], order[b].L.I[2])] = b;
  }
  auto lookup = [&](int level, const int P[3]) -> int {
    auto it = g.index.find(pack(level, P[0], P[1], P[2]));
    return it == g.index.end() ? -1 : it->second;
  };
  // block at or above position P of `level`; -1 if P is covered by finer blocks
  auto containing = [&](int level, const int P[3], int* found_level) -> int {
    for (int l = level; l >= 0; --l) {
      const int s = level - l;
      const int Q[3] = {P[0] >> s, P[1] >> s, P[2] >> s};
      const int id = lookup(l, Q);
      if (id >= 0) { *found_level = l; return id; }
    }
    return -1;
  };

  // ------------------------------------------------------------ neighbour table --
  g.nbr.assign((size_t)nB * 27 * 4, -1);
  g.dlev.assign((size_t)nB * 27, 0);
  for (int b = 0; b < nB; ++b) {
    const Leaf& L = g.leaf[b];
    for (int q = 0; q < 27; ++q) {
      const int d[3] = {q % 3 - 1, (q / 3) % 3 - 1, q / 9 - 1};
      int32_t* out = &g.nbr[((size_t)b * 27 + q) * 4];
      int P[3];
      if (!T.shifted(L, d, P)) { g.dlev[(size_t)b * 27 + q] = -100; continue; }
      int fl;
      const int id = containing(L.level, P, &fl);
      if (id >= 0) {
        g.dlev[(size_t)b * 27 + q] = (int8_t)(L.level - fl);
        out[0] = id;
        continue;
      }
      g.dlev[(size_t)b * 27 + q] = -1;          // finer: the children of P that touch b
      int n = 0;
      for (int o = 0; o < 8; ++o) {             // lower tangential axis fastest
        const int oo[3] = {o & 1, (o >> 1) & 1, o >> 2};
        bool touches = true;
        for (int a = 0; a < 3; ++a)
          if ((d[a] == 1 && oo[a] != 0) || (d[a] == -1 && oo[a] != 1)) touches = false;
        if (!touches) continue;
        const int F[3] = {2 * P[0] + oo[0], 2 * P[1] + oo[1], 2 * P[2] + oo[2]};
        out[n++] = lookup(L.level + 1, F);
      }
    }
  }

  // --------------------------------------------------------------- ghost messages --
  // One record per (destination block, direction, source block).  Per axis the
  // destination cells are {-2,-1} / {0..7} / {8,9}; the source cell is an affine
  // map of the destination cell followed by a shift (see batl_ghost_msg).
  g.msg.clear();
  g.msg_start.assign(nB + 1, 0);
  for (int b = 0; b < nB; ++b) {
    const Leaf& L = g.leaf[b];
    g.msg_start[b] = (int32_t)g.msg.size();
    for (int q = 0; q < 27; ++q) {
      if (q == 13) continue;
      const int d[3] = {q % 3 - 1, (q / 3) % 3 - 1, q / 9 - 1};
      batl_ghost_msg m{};
      m.dst = b;
      m.dir = (int8_t)q;
      for (int a = 0; a < 3; ++a) {
        m.lo[a] = (int8_t)(d[a] < 0 ? -NG : d[a] > 0 ? NI : 0);
        m.n[a] = (int8_t)(d[a] == 0 ? NI : NG);
      }
      // boundary handling per axis (Q-G5): periodic wraps, float clamps the cell
      // coordinate into the domain, fixed takes the prescribed state (lowest face wins)
      int P[3], de[3];
      bool clamp[3] = {false, false, false};
      int clamp_cell[3] = {0, 0, 0};
      int fixed_face = -1;
      for (int a = 0; a < 3; ++a) {
        const int N = cfg.n_root[a] << L.level;
        de[a] = d[a];
        P[a] = L.I[a] + d[a];
        if (P[a] < 0 || P[a] >= N) {
          const int face = 2 * a + (P[a] >= N ? 1 : 0);
          if (cfg.bc[face] == BATL_BC_PERIODIC) P[a] = (P[a] + N) % N;
          else if (cfg.bc[face] == BATL_BC_FIXED) { if (fixed_face < 0) fixed_face = face; }
          else { clamp[a] = true; clamp_cell[a] = d[a] < 0 ? 0 : NI - 1; de[a] = 0; P[a] = L.I[a]; }
        }
      }
      if (fixed_face >= 0) {
        m.kind = BATL_MSG_FIXED;
        m.src = -2 - fixed_face;
        g.msg.push_back(m);
        continue;
      }
      int fl = L.level;
      const int id = (de[0] == 0 && de[1] == 0 && de[2] == 0) ? b : containing(L.level, P, &fl);
      if (id >= 0 && fl == L.level) {                    // same level (or the block itself)
        m.kind = BATL_MSG_COPY;
        m.src = id;
        for (int a = 0; a < 3; ++a) {
          if (clamp[a]) { m.mul[a] = 0; m.off[a] = (int8_t)clamp_cell[a]; }
          else { m.mul[a] = 1; m.off[a] = (int8_t)(-NI * de[a]); }
          m.shift[a] = 0;
        }
        g.msg.push_back(m);
      } else if (id >= 0) {                              // coarser: first-order prolongation (Q-G4)
        if (fl != L.level - 1) { err = "grid not properly nested"; return BATL_EGRID; }
        m.kind = BATL_MSG_PROLONG;
        m.src = id;
        for (int a = 0; a < 3; ++a) {
          const int half = NI * (P[a] & 1);              // which half of the coarse block
          if (clamp[a]) { m.mul[a] = 0; m.off[a] = (int8_t)((clamp_cell[a] + half) >> 1); m.shift[a] = 0; }
          else { m.mul[a] = 1; m.off[a] = (int8_t)(half - NI * de[a]); m.shift[a] = 1; }
        }
        g.msg.push_back(m);
      } else {                                           // finer: one record per fine source block
        m.kind = BATL_MSG_RESTRICT;
        int nsub[3];
        for (int a = 0; a < 3; ++a) nsub[a] = (de[a] == 0 && !clamp[a]) ? 2 : 1;
        for (int s2 = 0; s2 < nsub[2]; ++s2)
          for (int s1 = 0; s1 < nsub[1]; ++s1)
            for (int s0 = 0; s0 < nsub[0]; ++s0) {
              const int sub[3] = {s0, s1, s2};
              batl_ghost_msg r = m;
              int F[3];
              for (int a = 0; a < 3; ++a) {
                if (clamp[a]) {                           // constant fine cell 2*(clamped cell)
                  F[a] = 2 * P[a] + (clamp_cell[a] >> 2);
                  r.mul[a] = 0; r.off[a] = (int8_t)(2 * (clamp_cell[a] & 3)); r.shift[a] = 0;
                } else if (de[a] == 0) {                  // tangential: halves 0..3 and 4..7
                  F[a] = 2 * P[a] + sub[a];
                  r.lo[a] = (int8_t)(4 * sub[a]); r.n[a] = 4;
                  r.mul[a] = 2; r.off[a] = (int8_t)(-NI * sub[a]); r.shift[a] = 0;
                } else {                                  // normal: fine block adjacent to b
                  F[a] = 2 * P[a] + (de[a] < 0 ? 1 : 0);
                  r.mul[a] = 2; r.off[a] = (int8_t)(de[a] < 0 ? NI : -2 * NI); r.shift[a] = 0;
                }
              }
              r.src = lookup(L.level + 1, F);
              if (r.src < 0) { err = "grid not properly nested"; return BATL_EGRID; }
              g.msg.push_back(r);
            }
      }
    }
  }
  g.msg_start[nB] = (int32_t)g.msg.size();

  // ------------------------------------------------------------ per-cell ghost plan --
  // The messages expanded to one entry per ghost cell (see batl_grid.hpp); identical
  // patterns are stored once.  Built once per grid like the paper's maps (L154-156).
  g.plan.clear();
  g.plan_id.assign(nB, -1);
  g.plan_src.assign((size_t)nB * PLAN_SLOTS, -1);
  {
    std::unordered_map<std::string, int32_t> seen;
    std::vector<uint32_t> cell(NCELL), pat(NGHOST);
    std::vector<uint8_t> covered(NCELL);
    for (int b = 0; b < nB; ++b) {
      std::fill(covered.begin(), covered.end(), 0);
      int32_t* slots = &g.plan_src[(size_t)b * PLAN_SLOTS];
      int n_slot = 0;
      for (int mi = g.msg_start[b]; mi < g.msg_start[b + 1]; ++mi) {
        const batl_ghost_msg& m = g.msg[mi];
        uint32_t slot = 0, kind = PLAN_FIXED;
        const bool prolong2 = m.kind == BATL_MSG_PROLONG && g.cfg.prolong_order == 2;
        if (m.kind != BATL_MSG_FIXED) {
          kind = (m.kind == BATL_MSG_RESTRICT) ? PLAN_RESTRICT : PLAN_COPY;
          int s = 0;
          while (s < n_slot && slots[s] != m.src) ++s;
          if (s == n_slot) {
            if (n_slot == PLAN_SLOTS) { err = "too many source blocks for one block"; return BATL_EGRID; }
            slots[n_slot++] = m.src;
          }
          slot = (uint32_t)s;
        }
        for (int ck = m.lo[2]; ck < m.lo[2] + m.n[2]; ++ck)
          for (int cj = m.lo[1]; cj < m.lo[1] + m.n[1]; ++cj)
            for (int ci = m.lo[0]; ci < m.lo[0] + m.n[0]; ++ci) {
              const int sd = ((ck + NG) * NS + (cj + NG)) * NS + (ci + NG);
              uint32_t ss;
              if (m.kind == BATL_MSG_FIXED) ss = (uint32_t)(-2 - m.src);
              else {
                const int sk = (m.mul[2] * ck + m.off[2]) >> m.shift[2];
                const int sj = (m.mul[1] * cj + m.off[1]) >> m.shift[1];
                const int si = (m.mul[0] * ci + m.off[0]) >> m.shift[0];
                ss = (uint32_t)(((sk + NG) * NS + (sj + NG)) * NS + (si + NG));
              }
              if (covered[sd]) { err = "ghost cell written twice"; return BATL_EGRID; }
              covered[sd] = 1;
              uint32_t kd = kind;
              if (prolong2) {
                // Q-G4b: which child of the coarse cell this fine cell is, per axis = the parity of its
                // (wrapped or clamped) global coordinate: of mul c + off where the source index is
                // (mul c + off) >> 1, of the clamped cell (0 below, 7 above the domain) where mul = 0
                const int c3[3] = {ci, cj, ck};
                kd = PLAN_PROLONG2;
                for (int a = 0; a < 3; ++a) {
                  const int par = (m.mul[a] == 0) ? (m.lo[a] < 0 ? 0 : 1) : ((m.mul[a] * c3[a] + m.off[a]) & 1);
                  kd |= (uint32_t)par << a;
                }
              }
              cell[sd] = (uint32_t)sd | (ss << 11) | (slot << 22) | (kd << 28);
            }
      }
      int n = 0;
      for (int s = 0; s < NCELL; ++s) {
        const int si = s % NS, sj = (s / NS) % NS, sk = s / (NS * NS);
        const bool phys = si >= NG && si < NG + NI && sj >= NG && sj < NG + NI && sk >= NG && sk < NG + NI;
        if (phys) continue;
        if (!covered[s]) { err = "ghost cell not covered by any message"; return BATL_EGRID; }
        pat[n++] = cell[s];
      }
      const std::string key(reinterpret_cast<const char*>(pat.data()), NGHOST * sizeof(uint32_t));
      auto it = seen.find(key);
      if (it == seen.end()) {
        it = seen.emplace(key, (int32_t)(g.plan.size() / NGHOST)).first;
        g.plan.insert(g.plan.end(), pat.begin(), pat.end());
      }
      g.plan_id[b] = it->second;
    }
    // blocks with second-order prolonged ghost cells: the second pass of the fill runs on them
    g.list_prolong.clear();
    for (int b = 0; b < nB; ++b) {
      const uint32_t* P = &g.plan[(size_t)g.plan_id[b] * NGHOST];
      bool any = false;
      for (int n = 0; n < NGHOST && !any; ++n) any = (P[n] >> 28) >= PLAN_PROLONG2;
      if (any) g.list_prolong.push_back(b);
    }
  }

  // ------------------------------------------------------------- block geometry --
  g.geom.resize(nB);
  g.body_mask.clear();
  for (int b = 0; b < nB; ++b) {
    const Leaf& L = g.leaf[b];
    BlockGeom& G = g.geom[b];
    for (int a = 0; a < 3; ++a) {
      const double root = (cfg.xyz_max[a] - cfg.xyz_min[a]) / (NI * cfg.n_root[a]);
      G.D[a] = std::ldexp(root, -L.level);
      G.invD[a] = std::ldexp(1.0 / root, L.level);
      G.x0[a] = cfg.xyz_min[a] + (NI * L.I[a]) * G.D[a];
    }
    G.level = L.level;
    G.flags = 0;
    G.mask_slot = -1;
    G.pad = 0;
    if (cfg.use_body) {                                   // body cells: centre inside r_body (L391)
      uint32_t words[BODY_MASK_WORDS] = {0};
      bool any = false;
      for (int k = -NG; k < NI + NG; ++k)
        for (int j = -NG; j < NI + NG; ++j)
          for (int i = -NG; i < NI + NG; ++i) {
            const double x = G.x0[0] + (i + 0.5) * G.D[0];
            const double y = G.x0[1] + (j + 0.5) * G.D[1];
            const double z = G.x0[2] + (k + 0.5) * G.D[2];
            if (x * x + y * y + z * z < cfg.r_body * cfg.r_body) {
              const int s = ((k + NG) * NS + (j + NG)) * NS + (i + NG);
              words[s >> 5] |= 1u << (s & 31);
              any = true;
            }
          }
      if (any) {
        G.flags |= 1;
        G.mask_slot = (int32_t)(g.body_mask.size() / BODY_MASK_WORDS);
        g.body_mask.insert(g.body_mask.end(), words, words + BODY_MASK_WORDS);
      }
    }
  }

  // the fused stage kernel takes the blocks free of body cells, the general kernel the others
  g.list_plain.clear();
  g.list_body.clear();
  for (int b = 0; b < nB; ++b) (g.geom[b].flags & 1 ? g.list_body : g.list_plain).push_back(b);

  // push table and fill list (see batl_grid.hpp); face directions in the 27-direction numbering
  static const int FACE_DIR[6] = {12, 14, 10, 16, 4, 22};
  g.push_nbr.assign((size_t)nB * 6, -1);
  g.push_fine.clear();
  g.list_fill.clear();
  // first-order prolongation (Q-G4) can be pushed as well: the coarse block's stage kernel writes each cell of
  // its outermost layer into the 2 x 2 x 2 fine ghost cells it covers
  // (not with flux correction: the corrected coarse cells are the very ones that are prolonged)
  const bool push_prolong = g.cfg.prolong_order == 1 && !g.cfg.flux_correction;
  for (int b = 0; b < nB; ++b) {
    bool fill = false;
    for (int f = 0; f < 6; ++f) {
      const int dir = FACE_DIR[f];
      const int8_t dl = g.dlev[(size_t)b * 27 + dir];
      int32_t& pn = g.push_nbr[(size_t)b * 6 + f];
      if (dl == 0) pn = g.nbr[((size_t)b * 27 + dir) * 4];
      else if (dl == -1) {                                 // finer: their ghosts are pushed, ours (restriction) are filled
        if (push_prolong) {
          pn = -2 - (int32_t)(g.push_fine.size() / 4);
          for (int q = 0; q < 4; ++q) g.push_fine.push_back(g.nbr[((size_t)b * 27 + dir) * 4 + q]);
        }
        fill = true;
      } else if (dl == 1 && push_prolong) pn = PUSH_BY_COARSER;   // the coarser neighbour writes these ghosts
      else fill = true;                                    // boundary face (or second-order prolongation)
    }
    if (fill) g.list_fill.push_back(b);
  }

  // flux correction (Q-G6b): a slot of the face-flux buffer for every block face at a resolution change
  // (both sides), and for every face that borders finer blocks the record the correction kernel reads
  g.fc_slot.assign((size_t)nB * 6, -1);
  g.fc_list.clear();
  g.fc_group.clear();
  g.n_fc_slots = 0;
  if (g.cfg.flux_correction) {
    for (int b = 0; b < nB; ++b)
      for (int f = 0; f < 6; ++f) {
        const int8_t dl = g.dlev[(size_t)b * 27 + FACE_DIR[f]];
        if (dl == 1 || dl == -1) g.fc_slot[(size_t)b * 6 + f] = g.n_fc_slots++;
      }
    for (int b = 0; b < nB; ++b)
      for (int f = 0; f < 6; ++f) {
        if (g.dlev[(size_t)b * 27 + FACE_DIR[f]] != -1) continue;
        int32_t rec[8] = {b, f, g.fc_slot[(size_t)b * 6 + f], -1, -1, -1, -1, 0};
        for (int q = 0; q < 4; ++q) {                     // the four fine blocks, lower tangential axis fastest
          const int32_t fb = g.nbr[((size_t)b * 27 + FACE_DIR[f]) * 4 + q];
          if (fb < 0) { err = "grid not properly nested"; return BATL_EGRID; }
          rec[3 + q] = g.fc_slot[(size_t)fb * 6 + (f ^ 1)];
          if (rec[3 + q] < 0) { err = "flux-correction tables inconsistent"; return BATL_EGRID; }
        }
        if (g.fc_group.empty() || g.fc_list[8 * (size_t)g.fc_group[g.fc_group.size() - 2]] != b) {
          g.fc_group.push_back((int32_t)(g.fc_list.size() / 8));   // first record of this block
          g.fc_group.push_back(0);
        }
        g.fc_group.back()++;
        g.fc_list.insert(g.fc_list.end(), rec, rec + 8);
      }
  }

  // conserved form of the fixed boundary states (eq. 5)
  for (int f = 0; f < 6; ++f) {
    const double* W = cfg.bc_prim[f];
    double* U = g.bc_cons[f];
    U[0] = W[0];
    for (int a = 0; a < 3; ++a) { U[1 + a] = W[0] * W[1 + a]; U[4 + a] = W[4 + a]; }
    const double u2 = W[1] * W[1] + W[2] * W[2] + W[3] * W[3];
    const double b2 = W[4] * W[4] + W[5] * W[5] + W[6] * W[6];
    U[7] = W[7] / (cfg.gamma - 1.0) + 0.5 * W[0] * u2 + 0.5 * b2;
  }
  return BATL_OK;
}

void expand_ghost_list(const HostGrid& g, std::vector<int32_t>& out) {
  struct Row { int32_t v[9]; };
  std::vector<Row> rows;
  rows.reserve(g.msg.size() * 64);
  for (const batl_ghost_msg& m : g.msg) {
    for (int ck = m.lo[2]; ck < m.lo[2] + m.n[2]; ++ck)
      for (int cj = m.lo[1]; cj < m.lo[1] + m.n[1]; ++cj)
        for (int ci = m.lo[0]; ci < m.lo[0] + m.n[0]; ++ci) {
          Row r;
          r.v[0] = m.dst; r.v[1] = ck; r.v[2] = cj; r.v[3] = ci; r.v[4] = m.kind; r.v[5] = m.src;
          if (m.kind == BATL_MSG_FIXED) { r.v[6] = r.v[7] = r.v[8] = 0; }
          else {
            r.v[6] = (m.mul[2] * ck + m.off[2]) >> m.shift[2];
            r.v[7] = (m.mul[1] * cj + m.off[1]) >> m.shift[1];
            r.v[8] = (m.mul[0] * ci + m.off[0]) >> m.shift[0];
          }
          rows.push_back(r);
        }
  }
  std::sort(rows.begin(), rows.end(), [](const Row& a, const Row& b) {
    for (int q = 0; q < 4; ++q) if (a.v[q] != b.v[q]) return a.v[q] < b.v[q];
    return false;
  });
  out.resize(rows.size() * 9);
  for (size_t r = 0; r < rows.size(); ++r) std::copy(rows[r].v, rows[r].v + 9, &out[9 * r]);
}

// The same canonical tuples, decoded from the per-cell plan the product kernel reads.
void expand_plan_list(const HostGrid& g, std::vector<int32_t>& out) {
  const int nB = g.n_blocks();
  out.clear();
  out.reserve((size_t)nB * NGHOST * 9);
  for (int b = 0; b < nB; ++b) {
    const uint32_t* P = &g.plan[(size_t)g.plan_id[b] * NGHOST];
    for (int n = 0; n < NGHOST; ++n) {          // storage order = (k, j, i) lexicographic
      const uint32_t e = P[n];
      const int sd = e & 2047, ss = (e >> 11) & 2047, slot = (e >> 22) & 63, kind = e >> 28;
      const int32_t src = g.plan_src[(size_t)b * PLAN_SLOTS + slot];
      int32_t row[9] = {b, sd / (NS * NS) - NG, (sd / NS) % NS - NG, sd % NS - NG, 0, 0, 0, 0, 0};
      if (kind == PLAN_FIXED) { row[4] = BATL_MSG_FIXED; row[5] = -2 - ss; }
      else {
        row[5] = src;
        row[6] = ss / (NS * NS) - NG; row[7] = (ss / NS) % NS - NG; row[8] = ss % NS - NG;
        if (kind == PLAN_RESTRICT) row[4] = BATL_MSG_RESTRICT;
        else if (kind >= PLAN_PROLONG2) row[4] = BATL_MSG_PROLONG;
        else row[4] = (g.leaf[src].level < g.leaf[b].level) ? BATL_MSG_PROLONG : BATL_MSG_COPY;
      }
      out.insert(out.end(), row, row + 9);
    }
  }
}

}  // namespace batl
