// ============================================================================
// mhd_oracle.cpp -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, obviously-correct CPU implementation (fp64) of the hot path of
// arXiv 2501.06717 ("BATSRUS GPU"): one explicit two-stage ideal-MHD step on a
// block-adaptive Cartesian grid.  Only tests/, __graft_entry__.smoke() and
// bench.py's cpu_baseline / --impl reference legs may build, load or call it.
// It shares no code, header, table or helper with paper_2501_06717_b200/ (the
// CUDA path) and neither includes the other.
//
// Structure follows PAPER.md Algorithm 1 (L29-64): per block
//   face values -> face fluxes -> source -> update, then exchange_messages
// with per-block scratch arrays (LeftState/RightState, Flux_V[XYZ], Source_VC).
// Ghost fill is brute force per ghost cell (no lists, no messages).
// Where the paper is silent the readings Q-* of SURVEY.md 8(c) are used; each
// is restated in DESIGN.md.  Citations "L<n>" are PAPER.md line numbers.
//
// Pins (tests/test_oracle_*.py, all -m "not gpu"):
//   grid      : leaf counts 15/120 (Table 2), 352 (config 3), closed
//               form periodic neighbours, hand enumeration on 2x1x1
//   ghost fill: L115 worked example, L146 message sizes, hand-computed
//               restriction/prolongation values, uniform state bit-identical
//   limiter   : linear data exact, zero at extrema, symmetry, TVD bound
//   flux      : F^(W,W)=F(W); eqs (1)-(4) term by term; c_s/c_A/c_F =
//               0.03/0.04/0.05 (L341); Sod vs exact Riemann solution
//   B0 split  : uniform-B0 equivalence; static dipole preserved bit-identically
//   update    : conservation to round-off; Alfven-wave 2nd-order convergence;
//               reflection symmetry bit-for-bit
//   sources   : Powell signs, Q-S2 and the B0 evaluation points, Q-T2/Q-T3, body
//               faces (tests/test_oracle_sources.py: closed forms and cancellations)
//   AMR       : second-order prolongation Q-G4b (linear field exact, children
//               average to the coarse cell, bounds) and flux correction Q-G6b
//               (totals conserved on the periodic AMR grid, closed-form corrected
//               cell) (tests/test_oracle_amr.py)
//   PARITY UNPINNED as readings of the paper (nothing in it decides them; each is
//   pinned as what DESIGN.md says it is): first- vs second-order prolongation
//   (Q-G4 / Q-G4b), flux correction or none (Q-G6 / Q-G6b), the name "Linde" (Q-F4).
// ============================================================================
#include <algorithm>
#include <array>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <map>
#include <set>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

constexpr int NI = 8;               // n_I = n_J = n_K (L391)
constexpr int NG = 2;               // ghost width n_G (L113)
constexpr int NS = NI + 2 * NG;     // stored cells per axis
constexpr int NV = 8;               // n_V
constexpr int NCELL = NS * NS * NS; // 1728 stored cells per block and variable

typedef std::array<int, 4> Key;     // (level, I, J, K)

struct Region { int shape, level; double p[6]; };

struct Oracle {
  int n_root[3];
  double lo[3], hi[3];
  int bc[6];
  double bc_prim[6][NV];
  std::vector<Region> regions;
  int max_level;
  double gamma, cfl, beta;
  int n_stage = 2;                  // 2: two-stage scheme (Q-U1); 1: one-stage, first order in time (L391-397)
  int flux_type = 0;                // 0 Rusanov (Q-F1), 1 HLL-type "Linde" flux (L343, Q-F4)
  int n_order = 2;                  // 2: limited linear reconstruction; 1: piecewise-constant face states (L86 nOrder)
  int prolong_order = 1;            // 1: Q-G4 (coarse value); 2: Q-G4b (limited linear profile of the coarse cell, two passes)
  int flux_corr = 0;                // 1: Q-G6b, coarse face flux at a resolution change := mean of the 4 fine face fluxes
  int dt_mode;                      // 0 global (lagged), 1 local, 2 fixed
  double dt_fixed;
  int use_divb, use_b0;
  double m[3];
  double lin_c[3] = {0, 0, 0};      // TEST-ONLY linear background field B0 = lin_c + lin_g x (use_b0 = 3)
  double lin_g[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
  int use_body;
  double r_body, rho_body, p_body;

  std::vector<Key> leaf;            // Morton order (Q-O1)
  std::map<Key, int> where;         // (level,I,J,K) -> block id
  std::vector<double> A, B;         // State_VGB twice: [block][var][k][j][i], 12^3 per var
  std::vector<double> dtc;          // local time step per physical cell [block][k][j][i]
  double t = 0.0;
  double dt_next = -1.0;            // < 0: no lagged dt available yet
  int warn = 0;
};

inline int sidx(int i, int j, int k) {      // i,j,k in [-2, 10)
  return ((k + NG) * NS + (j + NG)) * NS + (i + NG);
}
inline size_t at(int b, int v, int i, int j, int k) {
  return ((size_t)b * NV + v) * NCELL + sidx(i, j, k);
}

// ---------------------------------------------------------------- geometry --
inline double block_size(const Oracle& o, int a, int level) {   // edge length of a block
  return std::ldexp((o.hi[a] - o.lo[a]) / o.n_root[a], -level);
}
inline double cell_size(const Oracle& o, int a, int level) {    // D_a
  return std::ldexp((o.hi[a] - o.lo[a]) / (NI * o.n_root[a]), -level);
}
inline double inv_cell_size(const Oracle& o, int a, int level) { // 1/D_a, exact power-of-2 scaling
  return std::ldexp(1.0 / ((o.hi[a] - o.lo[a]) / (NI * o.n_root[a])), level);
}

// O-1: does the block box intersect the refinement region?
bool intersects(const Oracle& o, const Key& L, const Region& r) {
  double blo[3], bhi[3];
  for (int a = 0; a < 3; ++a) {
    double s = block_size(o, a, L[0]);
    blo[a] = o.lo[a] + L[1 + a] * s;
    bhi[a] = o.lo[a] + (L[1 + a] + 1) * s;
  }
  if (r.shape == 0) return true;
  if (r.shape == 1) {               // open box (p0..2 = lo, p3..5 = hi)
    for (int a = 0; a < 3; ++a)
      if (!(blo[a] < r.p[3 + a] && bhi[a] > r.p[a])) return false;
    return true;
  }
  double d2 = 0.0;                  // sphere: p0..2 centre, p3 radius
  for (int a = 0; a < 3; ++a) {
    double c = r.p[a], d = 0.0;
    if (c < blo[a]) d = blo[a] - c;
    else if (c > bhi[a]) d = c - bhi[a];
    d2 += d * d;
  }
  return d2 < r.p[3] * r.p[3];
}

void refine(std::set<Key>& leaves, const Key& L) {
  leaves.erase(L);
  for (int oz = 0; oz < 2; ++oz)
    for (int oy = 0; oy < 2; ++oy)
      for (int ox = 0; ox < 2; ++ox)
        leaves.insert(Key{L[0] + 1, 2 * L[1] + ox, 2 * L[2] + oy, 2 * L[3] + oz});
}

// O-1 / Q-O1 / Q-O2: roots, region refinement, 2:1 nesting, Morton order.
void build_grid(Oracle& o) {
  std::set<Key> leaves;
  for (int k = 0; k < o.n_root[2]; ++k)
    for (int j = 0; j < o.n_root[1]; ++j)
      for (int i = 0; i < o.n_root[0]; ++i) leaves.insert(Key{0, i, j, k});

  bool changed = true;
  while (changed) {                 // refine by regions until stable
    changed = false;
    std::vector<Key> cur(leaves.begin(), leaves.end());
    for (const Key& L : cur)
      for (const Region& r : o.regions)
        if (L[0] < r.level && L[0] < o.max_level && intersects(o, L, r)) {
          refine(leaves, L);
          changed = true;
          break;
        }
  }

  // Q-O2: leaves touching across a face, edge or corner differ by <= 1 level.
  // Brute force over pairs, integer boxes at the finest level, periodic images.
  changed = true;
  while (changed) {
    changed = false;
    int lmin = 1 << 30, lmax = 0;
    for (const Key& L : leaves) { lmin = std::min(lmin, L[0]); lmax = std::max(lmax, L[0]); }
    if (lmax - lmin < 2) break;
    std::vector<Key> cur(leaves.begin(), leaves.end());
    std::vector<char> mark(cur.size(), 0);
    for (size_t x = 0; x < cur.size(); ++x) {
      const Key& a = cur[x];
      for (size_t y = 0; y < cur.size() && !mark[x]; ++y) {
        const Key& b = cur[y];
        if (b[0] < a[0] + 2) continue;
        bool touch = true;
        for (int ax = 0; ax < 3 && touch; ++ax) {
          long N = (long)o.n_root[ax] << lmax;
          long a0 = (long)a[1 + ax] << (lmax - a[0]), a1 = (long)(a[1 + ax] + 1) << (lmax - a[0]);
          long b0 = (long)b[1 + ax] << (lmax - b[0]), b1 = (long)(b[1 + ax] + 1) << (lmax - b[0]);
          bool per = (o.bc[2 * ax] == 0);
          bool ok = false;
          for (int s = -1; s <= 1; ++s) {
            if (s != 0 && !per) continue;
            if (a0 <= b1 + s * N && b0 + s * N <= a1) ok = true;
          }
          touch = ok;
        }
        if (touch) mark[x] = 1;
      }
    }
    for (size_t x = 0; x < cur.size(); ++x)
      if (mark[x]) { refine(leaves, cur[x]); changed = true; }
  }

  // Q-O1: Morton order = (root index, child digits from the top level down).
  std::vector<std::pair<std::vector<int>, Key>> keyed;
  for (const Key& L : leaves) {
    int lev = L[0];
    int r[3] = {L[1] >> lev, L[2] >> lev, L[3] >> lev};
    std::vector<int> key;
    key.push_back(r[0] + o.n_root[0] * (r[1] + o.n_root[1] * r[2]));
    for (int l = 1; l <= lev; ++l) {
      int sh = lev - l;
      key.push_back(((L[1] >> sh) & 1) + 2 * ((L[2] >> sh) & 1) + 4 * ((L[3] >> sh) & 1));
    }
    keyed.push_back({key, L});
  }
  std::sort(keyed.begin(), keyed.end());
  o.leaf.clear();
  o.where.clear();
  for (auto& kv : keyed) {
    o.where[kv.second] = (int)o.leaf.size();
    o.leaf.push_back(kv.second);
  }
  size_t n = o.leaf.size() * (size_t)NV * NCELL;
  o.A.assign(n, 0.0);
  o.B.assign(n, 0.0);
  o.dtc.assign(o.leaf.size() * (size_t)NI * NI * NI, 0.0);
}

// leaf containing block position P at `level`: returns id and its level, or -1
// if the position is subdivided further (leaves are finer).
int find_leaf(const Oracle& o, int level, const int P[3], int* found_level) {
  for (int l = level; l >= 0; --l) {
    int s = level - l;
    auto it = o.where.find(Key{l, P[0] >> s, P[1] >> s, P[2] >> s});
    if (it != o.where.end()) { *found_level = l; return it->second; }
  }
  return -1;
}

// 8(b) table formats: dir = (di+1)+3(dj+1)+9(dk+1); dlev 0 same, +1 coarser,
// -1 finer, -100 outside a non-periodic boundary.
void neighbors(const Oracle& o, int32_t* nbr, int8_t* dlev) {
  int nB = (int)o.leaf.size();
  for (int b = 0; b < nB; ++b) {
    const Key& L = o.leaf[b];
    for (int dk = -1; dk <= 1; ++dk)
      for (int dj = -1; dj <= 1; ++dj)
        for (int di = -1; di <= 1; ++di) {
          int dir = (di + 1) + 3 * (dj + 1) + 9 * (dk + 1);
          int32_t* out = nbr + ((size_t)b * 27 + dir) * 4;
          out[0] = out[1] = out[2] = out[3] = -1;
          int d[3] = {di, dj, dk}, P[3];
          bool outside = false;
          for (int a = 0; a < 3; ++a) {
            int N = o.n_root[a] << L[0];
            P[a] = L[1 + a] + d[a];
            if (P[a] < 0 || P[a] >= N) {
              int face = 2 * a + (P[a] >= N ? 1 : 0);
              if (o.bc[face] == 0) P[a] = (P[a] + N) % N;
              else outside = true;
            }
          }
          if (outside) { dlev[b * 27 + dir] = -100; continue; }
          int fl;
          int id = find_leaf(o, L[0], P, &fl);
          if (id >= 0) {
            dlev[b * 27 + dir] = (int8_t)(L[0] - fl);      // 0 or +1
            out[0] = id;
            continue;
          }
          dlev[b * 27 + dir] = -1;                          // finer: children touching b
          int n = 0;
          for (int oz = 0; oz < 2; ++oz)
            for (int oy = 0; oy < 2; ++oy)
              for (int ox = 0; ox < 2; ++ox) {
                int oo[3] = {ox, oy, oz};
                bool ok = true;
                for (int a = 0; a < 3; ++a) {
                  if (d[a] == +1 && oo[a] != 0) ok = false;
                  if (d[a] == -1 && oo[a] != 1) ok = false;
                }
                if (!ok) continue;
                auto it = o.where.find(Key{L[0] + 1, 2 * P[0] + ox, 2 * P[1] + oy, 2 * P[2] + oz});
                out[n++] = (it == o.where.end()) ? -1 : it->second;
              }
        }
  }
}

// ------------------------------------------------------------- ghost fill --
// O-2 (L64, L113-117, L128, L146): where does ghost cell (i,j,k) of block b
// take its value from?  kind 0 copy, 1 restriction (src = lowest-index fine
// cell of the 8), 2 prolongation (first order, Q-G4), 3 fixed boundary state
// (src block = -2-face).
struct Src { int kind, sb, i, j, k; int par[3]; };   // par (prolongation): the fine cell is the low (0) / high (1) child along each axis

Src ghost_source(const Oracle& o, int b, int i, int j, int k) {
  const Key& L = o.leaf[b];
  int c[3] = {i, j, k}, g[3];
  int fixed_face = -1;
  for (int a = 0; a < 3; ++a) {
    int N = (NI * o.n_root[a]) << L[0];
    g[a] = NI * L[1 + a] + c[a];
    if (g[a] < 0 || g[a] >= N) {
      int face = 2 * a + (g[a] >= N ? 1 : 0);
      if (o.bc[face] == 0) g[a] = (g[a] + N) % N;          // periodic: wrap
      else if (o.bc[face] == 2) { if (fixed_face < 0) fixed_face = face; }  // lowest face wins
      else g[a] = (g[a] < 0) ? 0 : N - 1;                   // float: clamp (Q-G5)
    }
  }
  if (fixed_face >= 0) return Src{3, -2 - fixed_face, 0, 0, 0, {0, 0, 0}};
  int P[3] = {g[0] >> 3, g[1] >> 3, g[2] >> 3}, fl;
  int id = find_leaf(o, L[0], P, &fl);
  if (id >= 0 && fl == L[0]) return Src{0, id, g[0] & 7, g[1] & 7, g[2] & 7, {0, 0, 0}};
  if (id >= 0) {                                            // coarser leaf: cell floor(g/2)
    int h[3] = {g[0] >> 1, g[1] >> 1, g[2] >> 1};
    return Src{2, id, h[0] & 7, h[1] & 7, h[2] & 7, {g[0] & 1, g[1] & 1, g[2] & 1}};
  }
  int f[3] = {2 * g[0], 2 * g[1], 2 * g[2]};               // finer leaves: cells 2g+{0,1}^3
  auto it = o.where.find(Key{L[0] + 1, f[0] >> 3, f[1] >> 3, f[2] >> 3});
  return Src{1, it == o.where.end() ? -1 : it->second, f[0] & 7, f[1] & 7, f[2] & 7, {0, 0, 0}};
}

// Q-G3: mean of 8 children in fixed pairwise order (x pairs, then y, then z).
inline double restrict8(const double a[8]) {   // a[ox + 2 oy + 4 oz]
  return (((a[0] + a[1]) + (a[2] + a[3])) + ((a[4] + a[5]) + (a[6] + a[7]))) * 0.125;
}

void prim_to_cons(double gamma, const double W[NV], double U[NV]) {  // eq. (5)
  double rho = W[0];
  U[0] = rho;
  for (int a = 0; a < 3; ++a) U[1 + a] = rho * W[1 + a];
  for (int a = 0; a < 3; ++a) U[4 + a] = W[4 + a];
  double u2 = W[1] * W[1] + W[2] * W[2] + W[3] * W[3];
  double b2 = W[4] * W[4] + W[5] * W[5] + W[6] * W[6];
  U[7] = W[7] / (gamma - 1.0) + 0.5 * rho * u2 + 0.5 * b2;
}

void cons_to_prim(double gamma, const double U[NV], double W[NV]) {  // O-3
  double rho = U[0];
  W[0] = rho;
  for (int a = 0; a < 3; ++a) W[1 + a] = U[1 + a] / rho;
  for (int a = 0; a < 3; ++a) W[4 + a] = U[4 + a];
  double u2 = W[1] * W[1] + W[2] * W[2] + W[3] * W[3];
  double b2 = W[4] * W[4] + W[5] * W[5] + W[6] * W[6];
  W[7] = (gamma - 1.0) * (U[7] - 0.5 * rho * u2 - 0.5 * b2);
}

inline double mc_slope(double dm, double dp, double beta);

// O-2.  prolong_order = 2 (Q-G4b; the paper names the operation, L128, and is
// silent on its order): a fine ghost cell takes the value of the limited linear profile of the
// coarse cell that contains it, evaluated at the fine cell centre,
//   U = U_C + sum_d (+-1/4) s_d,   s_d = MC(beta)(U_C - U_{C-e_d}, U_{C+e_d} - U_C)   (O-4's limiter, per
// stored conserved variable, Q-G2; + for the high child along d, - for the low one; d = x, y, z in
// this order).  U_{C+-e_d} may be ghost cells of the coarse block, so the fill takes two passes:
// first everything that reads physical cells only (copy, restriction, boundary states), then the
// prolongation.  With the nesting rule Q-O2 no cell read in the second pass is itself prolonged.
void fill_ghosts(const Oracle& o, std::vector<double>& S) {
  int nB = (int)o.leaf.size();
  double Ufix[6][NV];
  for (int f = 0; f < 6; ++f) prim_to_cons(o.gamma, o.bc_prim[f], Ufix[f]);
#pragma omp parallel for schedule(static)
  for (int b = 0; b < nB; ++b)
    for (int k = -NG; k < NI + NG; ++k)
      for (int j = -NG; j < NI + NG; ++j)
        for (int i = -NG; i < NI + NG; ++i) {
          bool phys = (i >= 0 && i < NI && j >= 0 && j < NI && k >= 0 && k < NI);
          if (phys) continue;
          Src s = ghost_source(o, b, i, j, k);
          if (s.kind == 2 && o.prolong_order == 2) continue;          // second pass
          for (int v = 0; v < NV; ++v) {
            double val;
            if (s.kind == 0 || s.kind == 2) val = S[at(s.sb, v, s.i, s.j, s.k)];
            else if (s.kind == 3) val = Ufix[-2 - s.sb][v];
            else {
              double a[8];
              for (int oz = 0; oz < 2; ++oz)
                for (int oy = 0; oy < 2; ++oy)
                  for (int ox = 0; ox < 2; ++ox)
                    a[ox + 2 * oy + 4 * oz] = S[at(s.sb, v, s.i + ox, s.j + oy, s.k + oz)];
              val = restrict8(a);
            }
            S[at(b, v, i, j, k)] = val;
          }
        }
  if (o.prolong_order != 2) return;
#pragma omp parallel for schedule(static)
  for (int b = 0; b < nB; ++b)
    for (int k = -NG; k < NI + NG; ++k)
      for (int j = -NG; j < NI + NG; ++j)
        for (int i = -NG; i < NI + NG; ++i) {
          bool phys = (i >= 0 && i < NI && j >= 0 && j < NI && k >= 0 && k < NI);
          if (phys) continue;
          Src s = ghost_source(o, b, i, j, k);
          if (s.kind != 2) continue;
          for (int v = 0; v < NV; ++v) {
            const double c0 = S[at(s.sb, v, s.i, s.j, s.k)];
            const double sx = mc_slope(c0 - S[at(s.sb, v, s.i - 1, s.j, s.k)], S[at(s.sb, v, s.i + 1, s.j, s.k)] - c0, o.beta);
            const double sy = mc_slope(c0 - S[at(s.sb, v, s.i, s.j - 1, s.k)], S[at(s.sb, v, s.i, s.j + 1, s.k)] - c0, o.beta);
            const double sz = mc_slope(c0 - S[at(s.sb, v, s.i, s.j, s.k - 1)], S[at(s.sb, v, s.i, s.j, s.k + 1)] - c0, o.beta);
            double val = c0;
            val += (s.par[0] ? 0.25 : -0.25) * sx;
            val += (s.par[1] ? 0.25 : -0.25) * sy;
            val += (s.par[2] ? 0.25 : -0.25) * sz;
            S[at(b, v, i, j, k)] = val;
          }
        }
}

// Is any cell read by the second pass of the prolongation itself a prolonged ghost cell?  (It must
// not be: pins the claim above on the test grids.)  Returns the number of such reads.
int64_t prolong_reads_prolonged(const Oracle& o) {
  int64_t n = 0;
  int nB = (int)o.leaf.size();
  for (int b = 0; b < nB; ++b)
    for (int k = -NG; k < NI + NG; ++k)
      for (int j = -NG; j < NI + NG; ++j)
        for (int i = -NG; i < NI + NG; ++i) {
          if (i >= 0 && i < NI && j >= 0 && j < NI && k >= 0 && k < NI) continue;
          Src s = ghost_source(o, b, i, j, k);
          if (s.kind != 2) continue;
          for (int a = 0; a < 3; ++a)
            for (int sg = -1; sg <= 1; sg += 2) {
              int c[3] = {s.i, s.j, s.k};
              c[a] += sg;
              if (c[0] >= 0 && c[0] < NI && c[1] >= 0 && c[1] < NI && c[2] >= 0 && c[2] < NI) continue;
              if (ghost_source(o, s.sb, c[0], c[1], c[2]).kind == 2) ++n;
            }
        }
  return n;
}

// ------------------------------------------------------------------ physics --
// Q-R2: generalised MC(beta) slope from the two one-sided differences (O-4).
inline double mc_slope(double dm, double dp, double beta) {
  if (dm * dp <= 0.0) return 0.0;
  double s = std::min(std::min(beta * std::fabs(dm), beta * std::fabs(dp)), 0.5 * std::fabs(dm + dp));
  return dm > 0.0 ? s : -s;
}

// analytic dipole at the origin, B0 = (3 (m.x) x / r^2 - m) / r^3
void dipole_b0(const double m[3], const double x[3], double B0[3]) {
  double r2 = x[0] * x[0] + x[1] * x[1] + x[2] * x[2];
  if (r2 == 0.0) { B0[0] = B0[1] = B0[2] = 0.0; return; }
  double r = std::sqrt(r2), r3 = r2 * r;
  double md = m[0] * x[0] + m[1] * x[1] + m[2] * x[2];
  for (int a = 0; a < 3; ++a) B0[a] = (3.0 * md * x[a] / r2 - m[a]) / r3;
}

// B0 at a point: use_b0 = 1 dipole (the product's mode); use_b0 = 2 is a TEST-ONLY
// uniform field B0 = m, used to pin the B0 terms (uniform-B0 split equivalence, T11);
// use_b0 = 3 is a TEST-ONLY linear field B0_a = lin_c_a + sum_b lin_g_ab x_b: its discrete
// divergence and curl are exact and need not vanish, and its value tells where it was
// evaluated, which pins the signs of Q-S2 and the evaluation points (tests/test_oracle_sources.py).
inline void b0_at(const Oracle& o, const double x[3], double B0[3]) {
  if (o.use_b0 == 2) { B0[0] = o.m[0]; B0[1] = o.m[1]; B0[2] = o.m[2]; return; }
  if (o.use_b0 == 3) {
    for (int a = 0; a < 3; ++a)
      B0[a] = o.lin_c[a] + (o.lin_g[a][0] * x[0] + o.lin_g[a][1] * x[1] + o.lin_g[a][2] * x[2]);
    return;
  }
  dipole_b0(o.m, x, B0);
}

// O-5: physical flux F(W) through a face with normal e_d and U(W); eqs (1)-(4)
// (L170-177) with the B = B0 + B1 split of Q-B1 (B0f = 0 gives the paper's form).
void phys_flux(int d, const double W[NV], const double B0f[3], double gamma, double F[NV], double U[NV]) {
  double rho = W[0], p = W[7];
  const double* u = W + 1;
  const double* B1 = W + 4;
  double un = u[d], B1n = B1[d], B0n = B0f[d];
  double B1sq = B1[0] * B1[0] + B1[1] * B1[1] + B1[2] * B1[2];
  double B0B1 = B0f[0] * B1[0] + B0f[1] * B1[1] + B0f[2] * B1[2];
  double uB1 = u[0] * B1[0] + u[1] * B1[1] + u[2] * B1[2];
  double u2 = u[0] * u[0] + u[1] * u[1] + u[2] * u[2];
  double e = p / (gamma - 1.0) + 0.5 * rho * u2 + 0.5 * B1sq;          // eq. (5)
  double ptot = p + 0.5 * B1sq + B0B1;
  F[0] = rho * un;                                                       // eq. (1)
  for (int a = 0; a < 3; ++a)                                            // eq. (2)
    F[1 + a] = rho * un * u[a] - B1n * B1[a] - B0n * B1[a] - B1n * B0f[a];
  F[1 + d] += ptot;
  for (int a = 0; a < 3; ++a)                                            // eq. (3)
    F[4 + a] = un * (B1[a] + B0f[a]) - (B1n + B0n) * u[a];
  F[7] = un * (e + ptot) - uB1 * (B1n + B0n);                            // eq. (4)
  U[0] = rho;
  for (int a = 0; a < 3; ++a) U[1 + a] = rho * u[a];
  for (int a = 0; a < 3; ++a) U[4 + a] = B1[a];
  U[7] = e;
}

// O-5: Rusanov flux (Q-F1) with the speed from the mean face state (Q-F2); flux_type 1: the
// HLL-type two-wave flux ("Linde flux", reading Q-F4) with the bounds
// S_L = min(0, u_n - c_f), S_R = max(0, u_n + c_f) of the same mean state:
//   F = (S_R F_L - S_L F_R + S_L S_R (U_R - U_L)) / (S_R - S_L).
void face_flux(int d, const double WL[NV], const double WR[NV], const double B0f[3], double gamma,
               double F[NV], double* Bn, double* cmax, int flux_type = 0) {
  double FL[NV], FR[NV], UL[NV], UR[NV], Wb[NV];
  phys_flux(d, WL, B0f, gamma, FL, UL);
  phys_flux(d, WR, B0f, gamma, FR, UR);
  for (int v = 0; v < NV; ++v) Wb[v] = 0.5 * (WL[v] + WR[v]);
  double Bt[3] = {Wb[4] + B0f[0], Wb[5] + B0f[1], Wb[6] + B0f[2]};
  double a2 = gamma * Wb[7] / Wb[0];
  double b2 = (Bt[0] * Bt[0] + Bt[1] * Bt[1] + Bt[2] * Bt[2]) / Wb[0];
  double bn2 = Bt[d] * Bt[d] / Wb[0];
  double s = a2 + b2;
  double disc = s * s - 4.0 * a2 * bn2;
  if (disc < 0.0) disc = 0.0;
  double cf = std::sqrt(0.5 * (s + std::sqrt(disc)));
  double c = std::fabs(Wb[1 + d]) + cf;
  if (flux_type == 1) {
    double sl = std::min(0.0, Wb[1 + d] - cf), sr = std::max(0.0, Wb[1 + d] + cf);
    for (int v = 0; v < NV; ++v) F[v] = (sr * FL[v] - sl * FR[v] + sl * sr * (UR[v] - UL[v])) / (sr - sl);
  } else {
    for (int v = 0; v < NV; ++v) F[v] = 0.5 * (FL[v] + FR[v]) - 0.5 * c * (UR[v] - UL[v]);
  }
  *Bn = 0.5 * (WL[4 + d] + WR[4 + d]);
  *cmax = c;
}

// One pass over all blocks (Alg. 1 lines 4-9).  stage 0: speeds only (initial
// dt, Q-T2); stage 1: out = base + (1/2) dt R(in); stage 2: out = base + dt R(in);
// stage 3: the only stage of the one-stage scheme (Q-U2), out = base + dt R(in) with
// the local dt_c (Q-T3) taken from this very pass.
// Returns min over non-body physical cells of dt_c (O-8) in *dtmin.
void sweep(Oracle& o, int stage, const std::vector<double>& in, const std::vector<double>& base,
           std::vector<double>& out, double dt_global, double* dtmin_out, int* warn_out) {
  int nB = (int)o.leaf.size();
  double dtmin = std::numeric_limits<double>::infinity();
  int warn = 0;
  const double factor = (stage == 1) ? 0.5 : 1.0;
  // Q-G6b (flux_corr = 1; the paper calls its form "nearly conservative", L168,
  // and says nothing else): where a block face borders FINER blocks, the flux through each of its
  // face cells is replaced by the mean of the fluxes through the four fine faces that cover it,
  // taken from the fine blocks' own boundary faces, before the update (in every stage).  Then what
  // leaves the fine cells enters the coarse cell and the scheme conserves on AMR grids.  Plainly:
  // pass 0 computes the face fluxes of every block and keeps those of the six boundary faces,
  // pass 1 computes them again, substitutes, and updates.  B^_n (Q-S1) and c_max (O-8) stay as they are.
  static const int NFB = NI * NI;                       // faces of one block boundary face
  const bool corr = o.flux_corr && stage != 0;
  std::vector<double> FB(corr ? (size_t)nB * 6 * NV * NFB : 0);    // [b][2 d + side][v][t1][t2]
  for (int pass = corr ? 0 : 1; pass < 2; ++pass) {
#pragma omp parallel for schedule(static) reduction(min : dtmin) reduction(| : warn)
  for (int b = 0; b < nB; ++b) {
    const Key& L = o.leaf[b];
    double D[3], invD[3], x0[3];                 // x0 = coordinate of the low corner of cell 0
    for (int a = 0; a < 3; ++a) {
      D[a] = cell_size(o, a, L[0]);
      invD[a] = inv_cell_size(o, a, L[0]);
      x0[a] = o.lo[a] + (NI * L[1 + a]) * D[a];
    }
    // --- primitives of every stored cell, body flags (O-3, Q-F3)
    std::vector<double> W((size_t)NV * NCELL);
    std::vector<char> body(NCELL, 0);
    for (int k = -NG; k < NI + NG; ++k)
      for (int j = -NG; j < NI + NG; ++j)
        for (int i = -NG; i < NI + NG; ++i) {
          double U[NV], Wc[NV];
          for (int v = 0; v < NV; ++v) U[v] = in[at(b, v, i, j, k)];
          cons_to_prim(o.gamma, U, Wc);
          for (int v = 0; v < NV; ++v) W[(size_t)v * NCELL + sidx(i, j, k)] = Wc[v];
          if (o.use_body) {
            double x = x0[0] + (i + 0.5) * D[0], y = x0[1] + (j + 0.5) * D[1], z = x0[2] + (k + 0.5) * D[2];
            body[sidx(i, j, k)] = (x * x + y * y + z * z < o.r_body * o.r_body) ? 1 : 0;
          }
          bool phys = (i >= 0 && i < NI && j >= 0 && j < NI && k >= 0 && k < NI);
          if (phys && !body[sidx(i, j, k)]) {    // warning flags on the stage's input state
            if (!std::isfinite(Wc[0]) || !std::isfinite(Wc[7])) warn |= 1;
            if (Wc[0] <= 0.0 || Wc[7] <= 0.0) warn |= 2;
          }
        }
    // --- face values and face fluxes per direction (Alg. 1 lines 5-6)
    // Flux[d][v][f][t1][t2] with f = 0..8 the face between cells f-1 and f along d
    static const int NF = (NI + 1) * NI * NI;
    std::vector<double> Flux((size_t)3 * NV * NF), Bnf((size_t)3 * NF), Cf((size_t)3 * NF);
    std::vector<double> B0face(o.use_b0 ? (size_t)3 * 3 * NF : 0);
    for (int d = 0; d < 3; ++d) {
      int e1 = (d + 1) % 3, e2 = (d + 2) % 3;
      for (int t2 = 0; t2 < NI; ++t2)
        for (int t1 = 0; t1 < NI; ++t1)
          for (int f = 0; f <= NI; ++f) {
            int cL[3], cR[3], cm[3], cp[3];
            cL[d] = f - 1; cL[e1] = t1; cL[e2] = t2;
            cR[d] = f;     cR[e1] = t1; cR[e2] = t2;
            int iL = sidx(cL[0], cL[1], cL[2]), iR = sidx(cR[0], cR[1], cR[2]);
            double WL[NV], WR[NV];
            // limited slopes of the two cells adjacent to the face (O-4, Q-R1..3)
            for (int side = 0; side < 2; ++side) {
              const int* c = side == 0 ? cL : cR;
              for (int a = 0; a < 3; ++a) { cm[a] = c[a]; cp[a] = c[a]; }
              cm[d] -= 1; cp[d] += 1;
              int ic = sidx(c[0], c[1], c[2]), im = sidx(cm[0], cm[1], cm[2]), ip = sidx(cp[0], cp[1], cp[2]);
              bool nearbody = body[ic] || body[im] || body[ip];
              for (int v = 0; v < NV; ++v) {
                const double* Wv = &W[(size_t)v * NCELL];
                double s = (nearbody || o.n_order == 1) ? 0.0 : mc_slope(Wv[ic] - Wv[im], Wv[ip] - Wv[ic], o.beta);
                if (side == 0) WL[v] = Wv[ic] + 0.5 * s;   // W^L_{c+1/2}
                else           WR[v] = Wv[ic] - 0.5 * s;   // W^R_{c-1/2}
              }
            }
            double B0f[3] = {0, 0, 0};
            size_t fi = ((size_t)f * NI + t1) * NI + t2;
            if (o.use_b0) {
              double xf[3];
              xf[d] = x0[d] + f * D[d];
              xf[e1] = x0[e1] + (t1 + 0.5) * D[e1];
              xf[e2] = x0[e2] + (t2 + 0.5) * D[e2];
              b0_at(o, xf, B0f);
              for (int a = 0; a < 3; ++a) B0face[((size_t)d * 3 + a) * NF + fi] = B0f[a];
            }
            double F[NV] = {0, 0, 0, 0, 0, 0, 0, 0}, Bn = 0.0, c = 0.0;
            bool bL = body[iL], bR = body[iR];
            if (!(bL && bR)) {
              if (bL || bR) {                    // Q-F3: fixed-density reflective body state
                double* Wb = bL ? WL : WR;
                const double* Wt = bL ? WR : WL;
                Wb[0] = o.rho_body;
                for (int a = 0; a < 3; ++a) Wb[1 + a] = -Wt[1 + a];
                for (int a = 0; a < 3; ++a) Wb[4 + a] = Wt[4 + a];
                Wb[7] = (o.p_body > 0.0) ? o.p_body : Wt[7];
              }
              face_flux(d, WL, WR, B0f, o.gamma, F, &Bn, &c, o.flux_type);
            }
            for (int v = 0; v < NV; ++v) Flux[((size_t)d * NV + v) * NF + fi] = F[v];
            Bnf[(size_t)d * NF + fi] = Bn;
            Cf[(size_t)d * NF + fi] = c;
          }
    }
    if (pass == 0) {                                     // keep the fluxes of the six boundary faces
      for (int d = 0; d < 3; ++d)
        for (int side = 0; side < 2; ++side)
          for (int v = 0; v < NV; ++v)
            for (int t1 = 0; t1 < NI; ++t1)
              for (int t2 = 0; t2 < NI; ++t2)
                FB[((((size_t)b * 6 + 2 * d + side) * NV + v) * NI + t1) * NI + t2] =
                    Flux[((size_t)d * NV + v) * NF + ((size_t)(side ? NI : 0) * NI + t1) * NI + t2];
      continue;
    }
    if (corr) {
      for (int d = 0; d < 3; ++d) {
        const int e1 = (d + 1) % 3, e2 = (d + 2) % 3;
        for (int side = 0; side < 2; ++side) {
          // the neighbour position at the block's own level; wrap at periodic boundaries
          int P[3] = {L[1], L[2], L[3]};
          P[d] += side ? 1 : -1;
          const int N = o.n_root[d] << L[0];
          if (P[d] < 0 || P[d] >= N) {
            if (o.bc[2 * d + side] != 0) continue;       // domain boundary: no neighbour
            P[d] = (P[d] + N) % N;
          }
          int fl;
          if (find_leaf(o, L[0], P, &fl) >= 0) continue; // same level or coarser: nothing to substitute
          for (int t1 = 0; t1 < NI; ++t1)
            for (int t2 = 0; t2 < NI; ++t2) {
              // the fine block that covers this face cell, and its face on the opposite side
              int oc[3];
              oc[d] = side ? 0 : 1; oc[e1] = t1 / 4; oc[e2] = t2 / 4;
              auto it = o.where.find(Key{L[0] + 1, 2 * P[0] + oc[0], 2 * P[1] + oc[1], 2 * P[2] + oc[2]});
              if (it == o.where.end()) continue;         // cannot happen on a properly nested grid
              const int fb = it->second, fside = side ? 0 : 1;
              const int u1 = 2 * (t1 % 4), u2 = 2 * (t2 % 4);
              for (int v = 0; v < NV; ++v) {
                const double* F4 = &FB[(((size_t)fb * 6 + 2 * d + fside) * NV + v) * NFB];
                // mean of the four, pairs along the lower tangential axis first (as in Q-G3)
                double m;
                if (e1 < e2) m = ((F4[u1 * NI + u2] + F4[(u1 + 1) * NI + u2]) + (F4[u1 * NI + u2 + 1] + F4[(u1 + 1) * NI + u2 + 1])) * 0.25;
                else         m = ((F4[u1 * NI + u2] + F4[u1 * NI + u2 + 1]) + (F4[(u1 + 1) * NI + u2] + F4[(u1 + 1) * NI + u2 + 1])) * 0.25;
                Flux[((size_t)d * NV + v) * NF + ((size_t)(side ? NI : 0) * NI + t1) * NI + t2] = m;
              }
            }
        }
      }
    }
    // --- source, time step, update per physical cell (Alg. 1 lines 7-8)
    for (int k = 0; k < NI; ++k)
      for (int j = 0; j < NI; ++j)
        for (int i = 0; i < NI; ++i) {
          int ic = sidx(i, j, k);
          if (body[ic]) {
            if (stage != 0) for (int v = 0; v < NV; ++v) out[at(b, v, i, j, k)] = base[at(b, v, i, j, k)];
            continue;
          }
          int c[3] = {i, j, k};
          double R[NV] = {0, 0, 0, 0, 0, 0, 0, 0};
          double divB1 = 0.0, speed = 0.0;
          double divB0 = 0.0, dB0[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};   // dB0[a][d] = d B0_a / d x_d
          for (int d = 0; d < 3; ++d) {
            int e1 = (d + 1) % 3, e2 = (d + 2) % 3;
            size_t fm = ((size_t)c[d] * NI + c[e1]) * NI + c[e2];
            size_t fp = ((size_t)(c[d] + 1) * NI + c[e1]) * NI + c[e2];
            for (int v = 0; v < NV; ++v)
              R[v] -= (Flux[((size_t)d * NV + v) * NF + fp] - Flux[((size_t)d * NV + v) * NF + fm]) * invD[d];
            divB1 += (Bnf[(size_t)d * NF + fp] - Bnf[(size_t)d * NF + fm]) * invD[d];     // Q-S1
            speed += std::max(Cf[(size_t)d * NF + fm], Cf[(size_t)d * NF + fp]) * invD[d]; // Q-T1
            if (o.use_b0)
              for (int a = 0; a < 3; ++a)
                dB0[a][d] = (B0face[((size_t)d * 3 + a) * NF + fp] - B0face[((size_t)d * 3 + a) * NF + fm]) * invD[d];
          }
          const double u[3] = {W[(size_t)1 * NCELL + ic], W[(size_t)2 * NCELL + ic], W[(size_t)3 * NCELL + ic]};
          const double B1[3] = {W[(size_t)4 * NCELL + ic], W[(size_t)5 * NCELL + ic], W[(size_t)6 * NCELL + ic]};
          double B0c[3] = {0, 0, 0};
          if (o.use_b0) {
            double xc[3] = {x0[0] + (i + 0.5) * D[0], x0[1] + (j + 0.5) * D[1], x0[2] + (k + 0.5) * D[2]};
            b0_at(o, xc, B0c);
          }
          if (o.use_divb) {                                  // Powell source, RHS of eqs (2)-(4)
            double uB1 = u[0] * B1[0] + u[1] * B1[1] + u[2] * B1[2];
            for (int a = 0; a < 3; ++a) R[1 + a] -= (B1[a] + B0c[a]) * divB1;
            for (int a = 0; a < 3; ++a) R[4 + a] -= u[a] * divB1;
            R[7] -= uB1 * divB1;
          }
          if (o.use_b0) {                                    // Q-S2
            divB0 = dB0[0][0] + dB0[1][1] + dB0[2][2];
            double curl[3] = {dB0[2][1] - dB0[1][2], dB0[0][2] - dB0[2][0], dB0[1][0] - dB0[0][1]};
            double S[3];
            S[0] = -B1[0] * divB0 - (curl[1] * B1[2] - curl[2] * B1[1]);
            S[1] = -B1[1] * divB0 - (curl[2] * B1[0] - curl[0] * B1[2]);
            S[2] = -B1[2] * divB0 - (curl[0] * B1[1] - curl[1] * B1[0]);
            for (int a = 0; a < 3; ++a) R[1 + a] += S[a];
            R[7] += u[0] * S[0] + u[1] * S[1] + u[2] * S[2];
          }
          double dt_c = o.cfl / speed;                       // O-8
          if (dt_c < dtmin) dtmin = dt_c;
          if (stage == 0) continue;
          size_t ci = (((size_t)b * NI + k) * NI + j) * NI + i;
          double dt;
          if (o.dt_mode == 1) {                              // Q-T3
            if (stage == 1 || stage == 3) o.dtc[ci] = dt_c;
            dt = o.dtc[ci];
          } else dt = dt_global;
          for (int v = 0; v < NV; ++v)                       // O-7
            out[at(b, v, i, j, k)] = base[at(b, v, i, j, k)] + (factor * dt) * R[v];
        }
  }
  }   // pass
  *dtmin_out = dtmin;
  *warn_out |= warn;
}

int advance(Oracle& o, int n_steps, double* t, double* dt_last) {
  double dt = 0.0, dtmin;
  for (int s = 0; s < n_steps; ++s) {
    if (o.dt_mode == 0) {
      if (o.dt_next < 0.0) sweep(o, 0, o.A, o.A, o.B, 0.0, &o.dt_next, &o.warn);   // Q-T2, n = 0
      dt = o.dt_next;
    } else if (o.dt_mode == 2) dt = o.dt_fixed;
    if (o.n_stage == 1) {                                   // Q-U2: U^{n+1} = U^n + dt R(U^n)
      sweep(o, 3, o.A, o.A, o.B, dt, &dtmin, &o.warn);
      fill_ghosts(o, o.B);
      o.A.swap(o.B);
      if (o.dt_mode == 0) o.dt_next = dtmin;
      if (o.dt_mode != 1) o.t += dt;
      continue;
    }
    sweep(o, 1, o.A, o.A, o.B, dt, &dtmin, &o.warn);        // U* = U^n + dt/2 R(U^n)
    fill_ghosts(o, o.B);
    sweep(o, 2, o.B, o.A, o.A, dt, &dtmin, &o.warn);        // U^{n+1} = U^n + dt R(U*)
    fill_ghosts(o, o.A);
    if (o.dt_mode == 0) o.dt_next = dtmin;
    if (o.dt_mode != 1) o.t += dt;
  }
  if (t) *t = o.t;
  if (dt_last) *dt_last = dt;
  int w = o.warn;
  o.warn = 0;
  return w;
}

}  // namespace

// ============================================================ C interface ====
extern "C" {

void* orc_create(const int* n_root, const double* lo, const double* hi, const int* bc,
                 const double* bc_prim, int n_region, const int* region_shape_level,
                 const double* region_p, int max_level, double gamma, double cfl, double beta,
                 int dt_mode, double dt_fixed, int use_divb, int use_b0, const double* dipole_m,
                 int use_body, double r_body, double rho_body, double p_body) {
  Oracle* o = new Oracle();
  for (int a = 0; a < 3; ++a) { o->n_root[a] = n_root[a]; o->lo[a] = lo[a]; o->hi[a] = hi[a]; o->m[a] = dipole_m[a]; }
  for (int f = 0; f < 6; ++f) { o->bc[f] = bc[f]; for (int v = 0; v < NV; ++v) o->bc_prim[f][v] = bc_prim[f * NV + v]; }
  for (int r = 0; r < n_region; ++r) {
    Region R;
    R.shape = region_shape_level[2 * r];
    R.level = region_shape_level[2 * r + 1];
    for (int q = 0; q < 6; ++q) R.p[q] = region_p[6 * r + q];
    o->regions.push_back(R);
  }
  o->max_level = max_level; o->gamma = gamma; o->cfl = cfl; o->beta = beta;
  o->dt_mode = dt_mode; o->dt_fixed = dt_fixed; o->use_divb = use_divb; o->use_b0 = use_b0;
  o->use_body = use_body; o->r_body = r_body; o->rho_body = rho_body; o->p_body = p_body;
  build_grid(*o);
  return o;
}
// n_stage in {1, 2}, n_order in {1, 2} (L86, L391-397); the default is the two-stage second-order scheme
void orc_set_scheme(void* h, int n_stage, int n_order) {
  Oracle& o = *(Oracle*)h;
  o.n_stage = n_stage; o.n_order = n_order;
}
void orc_set_flux(void* h, int flux_type) { ((Oracle*)h)->flux_type = flux_type; }
// resolution changes: prolong_order in {1, 2} (Q-G4 / Q-G4b), flux_corr in {0, 1} (Q-G6 / Q-G6b);
// the defaults (1, 0) are the scheme of BASELINE.json's configs
void orc_set_amr(void* h, int prolong_order, int flux_corr) {
  Oracle& o = *(Oracle*)h;
  o.prolong_order = prolong_order; o.flux_corr = flux_corr;
}
int64_t orc_prolong_reads_prolonged(void* h) { return prolong_reads_prolonged(*(Oracle*)h); }
// TEST-ONLY: B0(x) = c + g x (g row-major [a][b] = dB0_a/dx_b); switches use_b0 to 3
void orc_set_b0_linear(void* h, const double* c, const double* g) {
  Oracle& o = *(Oracle*)h;
  o.use_b0 = 3;
  for (int a = 0; a < 3; ++a) { o.lin_c[a] = c[a]; for (int b = 0; b < 3; ++b) o.lin_g[a][b] = g[3 * a + b]; }
}
void orc_free(void* h) { delete (Oracle*)h; }
int orc_n_blocks(void* h) { return (int)((Oracle*)h)->leaf.size(); }
void orc_get_blocks(void* h, int32_t* out) {
  Oracle& o = *(Oracle*)h;
  for (size_t b = 0; b < o.leaf.size(); ++b) for (int q = 0; q < 4; ++q) out[4 * b + q] = o.leaf[b][q];
}
void orc_get_neighbors(void* h, int32_t* nbr, int8_t* dlev) { neighbors(*(Oracle*)h, nbr, dlev); }

// expanded canonical ghost list: (dst, k, j, i, kind, src, k', j', i') per ghost
// cell, block-major then k, j, i ascending (already lexicographically sorted).
int64_t orc_ghost_list(void* h, int32_t* out) {
  Oracle& o = *(Oracle*)h;
  int64_t n = 0;
  for (int b = 0; b < (int)o.leaf.size(); ++b)
    for (int k = -NG; k < NI + NG; ++k)
      for (int j = -NG; j < NI + NG; ++j)
        for (int i = -NG; i < NI + NG; ++i) {
          if (i >= 0 && i < NI && j >= 0 && j < NI && k >= 0 && k < NI) continue;
          if (out) {
            Src s = ghost_source(o, b, i, j, k);
            int32_t* r = out + 9 * n;
            r[0] = b; r[1] = k; r[2] = j; r[3] = i; r[4] = s.kind; r[5] = s.sb; r[6] = s.k; r[7] = s.j; r[8] = s.i;
          }
          ++n;
        }
  return n;
}

void orc_fill_ghosts(void* h) { Oracle& o = *(Oracle*)h; fill_ghosts(o, o.A); }

// physical cells only, [blk][var][k][j][i] with 8^3 per var; fills ghosts
void orc_set_state(void* h, const double* U) {
  Oracle& o = *(Oracle*)h;
  for (int b = 0; b < (int)o.leaf.size(); ++b)
    for (int v = 0; v < NV; ++v)
      for (int k = 0; k < NI; ++k) for (int j = 0; j < NI; ++j) for (int i = 0; i < NI; ++i)
        o.A[at(b, v, i, j, k)] = U[((((size_t)b * NV + v) * NI + k) * NI + j) * NI + i];
  fill_ghosts(o, o.A);
  o.t = 0.0; o.dt_next = -1.0; o.warn = 0;
}
void orc_set_primitive(void* h, const double* Win) {
  Oracle& o = *(Oracle*)h;
  for (int b = 0; b < (int)o.leaf.size(); ++b)
    for (int k = 0; k < NI; ++k) for (int j = 0; j < NI; ++j) for (int i = 0; i < NI; ++i) {
      double W[NV], U[NV];
      for (int v = 0; v < NV; ++v) W[v] = Win[((((size_t)b * NV + v) * NI + k) * NI + j) * NI + i];
      prim_to_cons(o.gamma, W, U);
      for (int v = 0; v < NV; ++v) o.A[at(b, v, i, j, k)] = U[v];
    }
  fill_ghosts(o, o.A);
  o.t = 0.0; o.dt_next = -1.0; o.warn = 0;
}
void orc_get_state(void* h, double* out, int with_ghost) {
  Oracle& o = *(Oracle*)h;
  if (with_ghost) { std::memcpy(out, o.A.data(), o.A.size() * sizeof(double)); return; }
  for (int b = 0; b < (int)o.leaf.size(); ++b)
    for (int v = 0; v < NV; ++v)
      for (int k = 0; k < NI; ++k) for (int j = 0; j < NI; ++j) for (int i = 0; i < NI; ++i)
        out[((((size_t)b * NV + v) * NI + k) * NI + j) * NI + i] = o.A[at(b, v, i, j, k)];
}
void orc_get_dt_local(void* h, double* out) {
  Oracle& o = *(Oracle*)h;
  std::memcpy(out, o.dtc.data(), o.dtc.size() * sizeof(double));
}
int orc_step(void* h, int n_steps, double* t, double* dt_last) { return advance(*(Oracle*)h, n_steps, t, dt_last); }

void orc_set_threads(int n) {
#ifdef _OPENMP
  omp_set_num_threads(n);
#else
  (void)n;
#endif
}
int orc_max_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

// ---- unit-level entry points for the pins -----------------------------------
double orc_mc_slope(double dm, double dp, double beta) { return mc_slope(dm, dp, beta); }
void orc_prim_to_cons(double gamma, const double* W, double* U) { prim_to_cons(gamma, W, U); }
void orc_cons_to_prim(double gamma, const double* U, double* W) { cons_to_prim(gamma, U, W); }
void orc_phys_flux(int d, const double* W, const double* B0f, double gamma, double* F, double* U) { phys_flux(d, W, B0f, gamma, F, U); }
void orc_face_flux(int d, const double* WL, const double* WR, const double* B0f, double gamma, double* F, double* Bn, double* cmax) {
  face_flux(d, WL, WR, B0f, gamma, F, Bn, cmax);
}
void orc_face_flux_type(int d, const double* WL, const double* WR, const double* B0f, double gamma, int flux_type,
                        double* F, double* Bn, double* cmax) {
  face_flux(d, WL, WR, B0f, gamma, F, Bn, cmax, flux_type);
}
void orc_dipole_b0(const double* m, const double* x, double* B0) { dipole_b0(m, x, B0); }
double orc_restrict8(const double* a) { return restrict8(a); }

}  // extern "C"
