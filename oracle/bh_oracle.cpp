// ORACLE — TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, obviously-correct CPU implementation of what the hot path of arxiv 1412.0659
// (Bedorf et al., "24.77 Pflops on a Gravitational Tree-Code ...") computes.  Only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may use it.
// It shares no code, header, table or constant generator with the CUDA library and neither
// includes the other.  Compile with -ffp-contract=off: no FMA is formed except where fma()/
// fmaf() is written.
//
// Two oracles:
//   O-direct : the definition.  Exact softened sum over all j != i in FP64
//              ("each of the N objects exerts N-1 interactions"; L184-190, Q = 0).
//   O-tree   : the Barnes-Hut algorithm step by step
//              with the readings T1..T12 / S1..S22 of SURVEY.md §8(c), restated in DESIGN.md.
//
// Pins (tests/test_oracle_*.py, all -m "not gpu"): two-body closed form, sum m a = 0,
// Plummer analytic potential, brute force in pure Python on tiny N, Hilbert bijection /
// adjacency / parent property, tree invariants, moments vs direct second moments, partition
// invariant of the walk, theta -> 0 == direct, p-c error ~ (size/distance)^3, a = grad phi,
// leapfrog circular orbit / reversibility.
// Option (not in PAPER.md): a second acceptance criterion, "bmax" (Salmon & Warren's bounding
// radius: accept iff D > b / theta, b = distance from the cell's centre of mass to the farthest corner of the TIGHT
// bounding box of its particles), selected with orc_tree_set_mac; the canonical criterion (S5) is the default and its
// arithmetic is untouched.  Pins: b bounds the distance of every particle of the cell from its c.o.m.; boxes nest.
// Option "relative" (SURVEY.md §8(f) NEXT-2 "per-group theta chosen to hit a force-error target", not in PAPER.md): an
// error-targeted criterion per group, selected with orc_tree_set_mac_relative(alpha, |a| per particle).  Group g accepts
// cell c iff the canonical criterion (S5, with the theta of the force call as a floor) accepts it AND
//     D^5 alpha a_g > M l^3,    a_g = the smallest given |a| among the group's particles,
// i.e. the first multipole term the evaluation leaves out, ~ M l^3 / D^5, stays below alpha times the group's own
// acceleration (the relative criterion of the tree-code literature, with the power that fits a quadrupole expansion).
// FP32, in this order: gscale = alpha * a_g; lhs = sqrt(D2) * D2 * D2 * gscale; q = M * l * l * l; accept iff lhs > q.
// Pins: alpha = 0 is direct summation; a huge alpha leaves the canonical lists; lists partition; monotone in alpha; the
// group's scale is the MINIMUM over its particles; lower cost than the canonical criterion at the same median error.
// Parity unpinned: the MAC formula itself (S5: PAPER.md L31 names an opening angle and defers to its ref. [9]) and the
// rounding order of T7 (S13: PAPER.md is silent on the precision of the moments) -- recorded readings, pinned only
// through their consequences (tree-vs-direct error, partition invariant, theta -> 0).
// Parity unpinned: the paper's interaction counts per particle (Table II) depend on
// group/MAC details and initial conditions that PAPER.md does not print; only their order of
// magnitude is comparable.
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <numeric>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

constexpr int KEY_BITS = 21;  // bits per dimension (S8): 63-bit key in a uint64

// ---------------------------------------------------------------- T3: Peano-Hilbert key
// Gray-code / rotation recurrence for n = 3 dimensions (PAPER.md L97 cites Hilbert keys [41];
// variant per SURVEY.md §8(c) T3).  Everything on 3-bit integers.
inline unsigned gc(unsigned i) { return i ^ (i >> 1); }
inline unsigned gc_inv(unsigned g) { return (g ^ (g >> 1) ^ (g >> 2)) & 7u; }
inline unsigned tsb(unsigned i) { unsigned n = 0; while (i & 1u) { ++n; i >>= 1; } return n; }
inline unsigned rotr3(unsigned x, unsigned k) { k %= 3; return ((x >> k) | (x << (3 - k))) & 7u; }
inline unsigned rotl3(unsigned x, unsigned k) { k %= 3; return ((x << k) | (x >> (3 - k))) & 7u; }
inline unsigned entry_pt(unsigned w) { return w == 0 ? 0u : gc(2u * ((w - 1u) / 2u)); }
inline unsigned dir_of(unsigned w) {
  if (w == 0) return 0u;
  return (w % 2u == 0) ? tsb(w - 1u) % 3u : tsb(w) % 3u;
}

uint64_t hilbert_key(uint32_t ix, uint32_t iy, uint32_t iz, int bits) {
  unsigned e = 0, d = 0;
  uint64_t h = 0;
  for (int b = bits - 1; b >= 0; --b) {
    unsigned l = (((iz >> b) & 1u) << 2) | (((iy >> b) & 1u) << 1) | ((ix >> b) & 1u);
    l = rotr3(l ^ e, d + 1);
    unsigned w = gc_inv(l);
    e = e ^ rotl3(entry_pt(w), d + 1);
    d = (d + dir_of(w) + 1) % 3;
    h = (h << 3) | w;
  }
  return h;
}

struct Cell {
  int32_t level;
  uint32_t first, count;
  int32_t first_child;  // -1 for a leaf
  int32_t n_child;
};

struct Tree {
  int64_t N = 0;
  int leaf_size = 16, group_size = 64;
  std::vector<float> pos, mass;        // caller order
  float lo[3], hi[3];                  // T1
  int k = 0;                           // side S = 2^k (T2)
  float origin[3];
  std::vector<uint64_t> key;           // caller order
  std::vector<uint32_t> order;         // sorted slot -> original index (T4)
  std::vector<uint64_t> skey;          // sorted keys
  std::vector<float> sx, sy, sz, sm;   // sorted-slot order
  std::vector<Cell> cells;             // BFS order (T5)
  std::vector<float> cM, cx, cy, cz, qxx, qyy, qzz, qxy, qxz, qyz, delta;  // T7, FP32 stored
  std::vector<float> tlo, thi, brad;   // option "bmax": tight box [n_cells][3] x 2 and bounding radius b about the c.o.m.
  int mac = 0;                         // 0: S5 (l / theta + delta), 1: bmax (b / theta), 2: relative (S5 as floor + D^5 alpha a_g > M l^3)
  std::vector<float> gscale;           // option "relative": alpha * min |a| of each group's particles
  std::vector<float> gmin, gmax;       // T8: [n_groups][3]
  std::vector<float> ropen2;           // T9, for the last theta
  std::vector<uint32_t> npp, npc;      // T10 per group
  int64_t n_groups() const { return (N + group_size - 1) / group_size; }
};

inline void grid_index(const Tree &t, const float *p, uint32_t out[3]) {
  // T2: one FP32 subtraction (the only rounding), exact power-of-two scale, floor, clamp.
  const float inv = std::ldexp(1.0f, KEY_BITS - t.k);
  for (int d = 0; d < 3; ++d) {
    float tt = p[d] - t.origin[d];
    float u = tt * inv;
    float f = std::floor(u);
    int64_t i = (f < 0.0f) ? 0 : (f >= 2097152.0f ? 2097151 : (int64_t)f);
    out[d] = (uint32_t)i;
  }
}

int build(Tree &t) {
  const int64_t N = t.N;
  // ---- T1 bbox
  for (int d = 0; d < 3; ++d) { t.lo[d] = std::numeric_limits<float>::infinity(); t.hi[d] = -t.lo[d]; }
  for (int64_t i = 0; i < N; ++i)
    for (int d = 0; d < 3; ++d) {
      float v = t.pos[3 * i + d];
      if (!std::isfinite(v)) return -5;
      t.lo[d] = std::min(t.lo[d], v);
      t.hi[d] = std::max(t.hi[d], v);
    }
  for (int64_t i = 0; i < N; ++i) if (!std::isfinite(t.mass[i])) return -5;
  // ---- T2 cube: centred on the bbox, side = smallest power of two > extent
  double ext = 0.0;
  for (int d = 0; d < 3; ++d) ext = std::max(ext, (double)t.hi[d] - (double)t.lo[d]);
  int k = 0;
  if (ext > 0.0) { int e; std::frexp(ext, &e); k = e; }  // ext = f 2^e, f in [0.5,1) => 2^e > ext >= 2^(e-1)
  t.k = k;
  const double S = std::ldexp(1.0, k);
  for (int d = 0; d < 3; ++d) {
    double c = 0.5 * ((double)t.lo[d] + (double)t.hi[d]);
    t.origin[d] = (float)(c - 0.5 * S);
  }
  // ---- T3 keys
  t.key.resize(N);
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < N; ++i) {
    uint32_t g[3];
    grid_index(t, &t.pos[3 * i], g);
    t.key[i] = hilbert_key(g[0], g[1], g[2], KEY_BITS);
  }
  // ---- T4 stable sort of the identity index array by key
  t.order.resize(N);
  std::iota(t.order.begin(), t.order.end(), 0u);
  std::stable_sort(t.order.begin(), t.order.end(),
                   [&](uint32_t a, uint32_t b) { return t.key[a] < t.key[b]; });
  t.skey.resize(N); t.sx.resize(N); t.sy.resize(N); t.sz.resize(N); t.sm.resize(N);
  for (int64_t s = 0; s < N; ++s) {
    uint32_t i = t.order[s];
    t.skey[s] = t.key[i];
    t.sx[s] = t.pos[3 * i]; t.sy[s] = t.pos[3 * i + 1]; t.sz[s] = t.pos[3 * i + 2];
    t.sm[s] = t.mass[i];
  }
  // ---- T5 octree: breadth-first; a cell is a leaf iff count <= leaf_size or
  // level == 21; children = maximal sub-runs sharing the next 3 key bits, in key order.
  t.cells.clear();
  t.cells.push_back(Cell{0, 0u, (uint32_t)N, -1, 0});
  for (size_t c = 0; c < t.cells.size(); ++c) {
    Cell cur = t.cells[c];
    if ((int64_t)cur.count <= t.leaf_size || cur.level == KEY_BITS) continue;
    const int shift = 3 * (KEY_BITS - 1 - cur.level);
    int32_t fc = (int32_t)t.cells.size();
    int nch = 0;
    uint32_t s = cur.first, end = cur.first + cur.count;
    while (s < end) {
      uint64_t dgt = (t.skey[s] >> shift) & 7u;
      uint32_t e = s + 1;
      while (e < end && ((t.skey[e] >> shift) & 7u) == dgt) ++e;
      t.cells.push_back(Cell{cur.level + 1, s, e - s, -1, 0});
      ++nch;
      s = e;
    }
    t.cells[c].first_child = fc;
    t.cells[c].n_child = nch;
  }
  // ---- T6 + T7 moments, bottom-up (BFS order reversed visits children before parents)
  const size_t nc = t.cells.size();
  t.cM.assign(nc, 0); t.cx.assign(nc, 0); t.cy.assign(nc, 0); t.cz.assign(nc, 0);
  t.qxx.assign(nc, 0); t.qyy.assign(nc, 0); t.qzz.assign(nc, 0);
  t.qxy.assign(nc, 0); t.qxz.assign(nc, 0); t.qyz.assign(nc, 0); t.delta.assign(nc, 0);
  for (size_t ci = nc; ci-- > 0;) {
    const Cell &c = t.cells[ci];
    double M = 0, s0 = 0, s1 = 0, s2 = 0;
    double Q[6] = {0, 0, 0, 0, 0, 0};
    float cf[3];
    if (c.first_child < 0) {
      for (uint32_t p = c.first; p < c.first + c.count; ++p) {
        double m = t.sm[p];
        M = M + m;
        s0 = s0 + m * (double)t.sx[p];
        s1 = s1 + m * (double)t.sy[p];
        s2 = s2 + m * (double)t.sz[p];
      }
      cf[0] = (float)(s0 / M); cf[1] = (float)(s1 / M); cf[2] = (float)(s2 / M);
      for (uint32_t p = c.first; p < c.first + c.count; ++p) {
        double m = t.sm[p];
        double dx = (double)t.sx[p] - (double)cf[0];
        double dy = (double)t.sy[p] - (double)cf[1];
        double dz = (double)t.sz[p] - (double)cf[2];
        double mx = m * dx, my = m * dy, mz = m * dz;
        Q[0] = Q[0] + mx * dx; Q[1] = Q[1] + my * dy; Q[2] = Q[2] + mz * dz;
        Q[3] = Q[3] + mx * dy; Q[4] = Q[4] + mx * dz; Q[5] = Q[5] + my * dz;
      }
    } else {
      for (int32_t ch = c.first_child; ch < c.first_child + c.n_child; ++ch) {
        double m = t.cM[ch];
        M = M + m;
        s0 = s0 + m * (double)t.cx[ch];
        s1 = s1 + m * (double)t.cy[ch];
        s2 = s2 + m * (double)t.cz[ch];
      }
      cf[0] = (float)(s0 / M); cf[1] = (float)(s1 / M); cf[2] = (float)(s2 / M);
      for (int32_t ch = c.first_child; ch < c.first_child + c.n_child; ++ch) {
        double m = t.cM[ch];
        double dx = (double)t.cx[ch] - (double)cf[0];
        double dy = (double)t.cy[ch] - (double)cf[1];
        double dz = (double)t.cz[ch] - (double)cf[2];
        double mx = m * dx, my = m * dy, mz = m * dz;
        Q[0] = Q[0] + ((double)t.qxx[ch] + mx * dx);
        Q[1] = Q[1] + ((double)t.qyy[ch] + my * dy);
        Q[2] = Q[2] + ((double)t.qzz[ch] + mz * dz);
        Q[3] = Q[3] + ((double)t.qxy[ch] + mx * dy);
        Q[4] = Q[4] + ((double)t.qxz[ch] + mx * dz);
        Q[5] = Q[5] + ((double)t.qyz[ch] + my * dz);
      }
    }
    // T6: geometric centre from the integer coordinates of the first particle
    const float pfirst[3] = {t.sx[c.first], t.sy[c.first], t.sz[c.first]};
    uint32_t g[3];
    grid_index(t, pfirst, g);
    const double lc = std::ldexp(1.0, t.k - c.level);
    double dd[3];
    for (int d = 0; d < 3; ++d) {
      double q = (double)(g[d] >> (KEY_BITS - c.level));
      double gc_ = (double)t.origin[d] + (q + 0.5) * lc;
      dd[d] = (double)cf[d] - gc_;
    }
    double del = std::sqrt((dd[0] * dd[0] + dd[1] * dd[1]) + dd[2] * dd[2]);
    t.cM[ci] = (float)M; t.cx[ci] = cf[0]; t.cy[ci] = cf[1]; t.cz[ci] = cf[2];
    t.qxx[ci] = (float)Q[0]; t.qyy[ci] = (float)Q[1]; t.qzz[ci] = (float)Q[2];
    t.qxy[ci] = (float)Q[3]; t.qxz[ci] = (float)Q[4]; t.qyz[ci] = (float)Q[5];
    t.delta[ci] = (float)del;
  }
  // ---- option "bmax": tight bounding box of every cell's particles, bottom-up (min / max are exact), and the
  // bounding radius about the FP32 centre of mass, FP32 in this order: e_d = max(c_d - lo_d, hi_d - c_d);
  // b2 = fma(e_z, e_z, fma(e_y, e_y, e_x * e_x)); b = sqrt(b2)
  t.tlo.assign(3 * nc, 0); t.thi.assign(3 * nc, 0); t.brad.assign(nc, 0);
  for (size_t ci = nc; ci-- > 0;) {
    const Cell &c = t.cells[ci];
    float lo[3], hi[3];
    for (int d = 0; d < 3; ++d) { lo[d] = std::numeric_limits<float>::infinity(); hi[d] = -lo[d]; }
    if (c.first_child < 0) {
      for (uint32_t p = c.first; p < c.first + c.count; ++p) {
        const float x[3] = {t.sx[p], t.sy[p], t.sz[p]};
        for (int d = 0; d < 3; ++d) { lo[d] = std::min(lo[d], x[d]); hi[d] = std::max(hi[d], x[d]); }
      }
    } else {
      for (int32_t ch = c.first_child; ch < c.first_child + c.n_child; ++ch)
        for (int d = 0; d < 3; ++d) { lo[d] = std::min(lo[d], t.tlo[3 * ch + d]); hi[d] = std::max(hi[d], t.thi[3 * ch + d]); }
    }
    const float cc[3] = {t.cx[ci], t.cy[ci], t.cz[ci]};
    float e[3];
    for (int d = 0; d < 3; ++d) {
      t.tlo[3 * ci + d] = lo[d]; t.thi[3 * ci + d] = hi[d];
      e[d] = std::max(cc[d] - lo[d], hi[d] - cc[d]);
    }
    const float b2 = std::fmaf(e[2], e[2], std::fmaf(e[1], e[1], e[0] * e[0]));
    t.brad[ci] = std::sqrt(b2);
  }
  // ---- T8 groups: fixed runs of group_size sorted slots, tight AABB
  const int64_t ng = t.n_groups();
  t.gmin.assign(3 * ng, 0); t.gmax.assign(3 * ng, 0);
  for (int64_t g = 0; g < ng; ++g) {
    int64_t a = g * t.group_size, b = std::min<int64_t>(a + t.group_size, N);
    float mn[3] = {t.sx[a], t.sy[a], t.sz[a]}, mx[3] = {t.sx[a], t.sy[a], t.sz[a]};
    for (int64_t s = a + 1; s < b; ++s) {
      mn[0] = std::min(mn[0], t.sx[s]); mx[0] = std::max(mx[0], t.sx[s]);
      mn[1] = std::min(mn[1], t.sy[s]); mx[1] = std::max(mx[1], t.sy[s]);
      mn[2] = std::min(mn[2], t.sz[s]); mx[2] = std::max(mx[2], t.sz[s]);
    }
    for (int d = 0; d < 3; ++d) { t.gmin[3 * g + d] = mn[d]; t.gmax[3 * g + d] = mx[d]; }
  }
  t.npp.assign(ng, 0); t.npc.assign(ng, 0);
  return 0;
}

// T9: opening radius squared, FP32, in this order: r = l_c / theta; r = r + delta; r*r.
void set_opening(Tree &t, float theta) {
  const size_t nc = t.cells.size();
  t.ropen2.resize(nc);
  for (size_t c = 0; c < nc; ++c) {
    if (t.mac == 1) {  // option "bmax": r = b / theta; r_open^2 = r * r
      float r = t.brad[c] / theta;
      if (theta == 0.0f) r = std::numeric_limits<float>::infinity();  // 0 / 0: theta = 0 still opens everything
      t.ropen2[c] = r * r;
      continue;
    }
    float lc = std::ldexp(1.0f, t.k - t.cells[c].level);
    float r = lc / theta;
    r = r + t.delta[c];
    t.ropen2[c] = r * r;
  }
}

// T10: multipole acceptance test of cell c against group g. true => accept (one p-c entry).
inline bool mac_accept(const Tree &t, int64_t g, int32_t c) {
  const float cc[3] = {t.cx[c], t.cy[c], t.cz[c]};
  float u[3];
  for (int d = 0; d < 3; ++d) {
    float a = t.gmin[3 * g + d] - cc[d];
    float b = cc[d] - t.gmax[3 * g + d];
    u[d] = std::max(0.0f, std::max(a, b));
  }
  float D2 = std::fmaf(u[2], u[2], std::fmaf(u[1], u[1], u[0] * u[0]));
  if (t.mac == 2) {  // option "relative": the canonical criterion as a floor, then D^5 alpha a_g > M l^3
    if (!(D2 > t.ropen2[c])) return false;
    float lc = std::ldexp(1.0f, t.k - t.cells[c].level);
    float lhs = std::sqrt(D2) * D2;
    lhs = lhs * D2;
    lhs = lhs * t.gscale[g];
    float q = t.cM[c] * lc;
    q = q * lc;
    q = q * lc;
    return lhs > q;
  }
  return D2 > t.ropen2[c];
}

// Walk of one group: collects accepted cells and opened leaves (T10).
void walk_group(const Tree &t, int64_t g, std::vector<int32_t> &acc_cells, std::vector<int32_t> &open_leaves) {
  std::vector<int32_t> stack;
  stack.push_back(0);
  while (!stack.empty()) {
    int32_t c = stack.back();
    stack.pop_back();
    if (mac_accept(t, g, c)) { acc_cells.push_back(c); continue; }
    const Cell &cl = t.cells[c];
    if (cl.first_child < 0) { open_leaves.push_back(c); continue; }
    for (int32_t ch = cl.first_child + cl.n_child - 1; ch >= cl.first_child; --ch) stack.push_back(ch);
  }
}

// T11: evaluation in FP64 from the FP32 inputs (Eqs. (1),(2) L186-188, softened per S1).
inline void eval_pp(double tx, double ty, double tz, double sx, double sy, double sz, double m,
                    double eps2, double a[3], double &phi) {
  double rx = sx - tx, ry = sy - ty, rz = sz - tz;
  double s2 = rx * rx + ry * ry + rz * rz + eps2;
  double rho = 1.0 / std::sqrt(s2);
  double rho3 = rho * rho * rho;
  phi -= m * rho;
  a[0] += m * rho3 * rx; a[1] += m * rho3 * ry; a[2] += m * rho3 * rz;
}

inline void eval_pc(const Tree &t, int32_t c, double tx, double ty, double tz, double eps2,
                    double a[3], double &phi) {
  double rx = (double)t.cx[c] - tx, ry = (double)t.cy[c] - ty, rz = (double)t.cz[c] - tz;
  double s2 = rx * rx + ry * ry + rz * rz + eps2;
  double rho = 1.0 / std::sqrt(s2);
  double rho2 = rho * rho, rho3 = rho2 * rho, rho5 = rho3 * rho2, rho7 = rho5 * rho2;
  double M = t.cM[c];
  double Qxx = t.qxx[c], Qyy = t.qyy[c], Qzz = t.qzz[c], Qxy = t.qxy[c], Qxz = t.qxz[c], Qyz = t.qyz[c];
  double T = Qxx + Qyy + Qzz;
  double vx = Qxx * rx + Qxy * ry + Qxz * rz;
  double vy = Qxy * rx + Qyy * ry + Qyz * rz;
  double vz = Qxz * rx + Qyz * ry + Qzz * rz;
  double q = rx * vx + ry * vy + rz * vz;
  phi += -M * rho + 0.5 * T * rho3 - 1.5 * q * rho5;
  double g = M * rho3 - 1.5 * T * rho5 + 7.5 * q * rho7;
  a[0] += g * rx - 3.0 * rho5 * vx;
  a[1] += g * ry - 3.0 * rho5 * vy;
  a[2] += g * rz - 3.0 * rho5 * vz;
}

// Tree force for groups g0, g0+stride, ... (stride 1 = all). Outputs in ORIGINAL particle order.
void tree_force(Tree &t, float theta, float eps, double *acc, double *pot, int64_t g0, int64_t stride) {
  set_opening(t, theta);
  const int64_t ng = t.n_groups();
  const double eps2 = (double)eps * (double)eps;
#pragma omp parallel
  {
    std::vector<int32_t> ac, ol;
#pragma omp for schedule(dynamic, 4)
    for (int64_t g = g0; g < ng; g += stride) {
      ac.clear(); ol.clear();
      walk_group(t, g, ac, ol);
      uint64_t pp = 0;
      for (int32_t c : ol) pp += t.cells[c].count;
      t.npp[g] = (uint32_t)pp;
      t.npc[g] = (uint32_t)ac.size();
      int64_t a0 = g * t.group_size, b0 = std::min<int64_t>(a0 + t.group_size, t.N);
      for (int64_t s = a0; s < b0; ++s) {
        double a[3] = {0, 0, 0}, phi = 0;
        double tx = t.sx[s], ty = t.sy[s], tz = t.sz[s];
        for (int32_t c : ol) {
          const Cell &cl = t.cells[c];
          for (uint32_t p = cl.first; p < cl.first + cl.count; ++p) {
            if ((int64_t)p == s) continue;  // S2: skip j == i by index
            eval_pp(tx, ty, tz, t.sx[p], t.sy[p], t.sz[p], t.sm[p], eps2, a, phi);
          }
        }
        for (int32_t c : ac) eval_pc(t, c, tx, ty, tz, eps2, a, phi);
        uint32_t i = t.order[s];
        if (acc) { acc[3 * (int64_t)i] = a[0]; acc[3 * (int64_t)i + 1] = a[1]; acc[3 * (int64_t)i + 2] = a[2]; }
        if (pot) pot[i] = phi;
      }
    }
  }
}

}  // namespace

// =============================================================================== C ABI
extern "C" {

uint64_t orc_hilbert_key(uint32_t ix, uint32_t iy, uint32_t iz, int bits) { return hilbert_key(ix, iy, iz, bits); }

int orc_num_threads() {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

// O-direct. targets == NULL => all particles (nt ignored). acc [nt][3], pot [nt], FP64.
int orc_direct(const float *pos, const float *mass, int64_t N, const int64_t *targets, int64_t nt,
               double eps, double *acc, double *pot) {
  if (!pos || !mass || N <= 0) return -1;
  if (!targets) nt = N;
  const double eps2 = eps * eps;
#pragma omp parallel for schedule(dynamic, 16)
  for (int64_t k = 0; k < nt; ++k) {
    int64_t i = targets ? targets[k] : k;
    double tx = pos[3 * i], ty = pos[3 * i + 1], tz = pos[3 * i + 2];
    double ax = 0, ay = 0, az = 0, phi = 0;
    for (int64_t j = 0; j < N; ++j) {
      if (j == i) continue;
      double rx = (double)pos[3 * j] - tx, ry = (double)pos[3 * j + 1] - ty, rz = (double)pos[3 * j + 2] - tz;
      double s2 = rx * rx + ry * ry + rz * rz + eps2;
      double rho = 1.0 / std::sqrt(s2);
      double m = mass[j];
      double mr3 = m * rho * rho * rho;
      phi -= m * rho;
      ax += mr3 * rx; ay += mr3 * ry; az += mr3 * rz;
    }
    if (acc) { acc[3 * k] = ax; acc[3 * k + 1] = ay; acc[3 * k + 2] = az; }
    if (pot) pot[k] = phi;
  }
  return 0;
}

// Single p-c evaluation (Eqs. (1),(2)) exposed for the pins: Q = {xx,yy,zz,xy,xz,yz}.
void orc_eval_pc(const double target[3], const float com[3], float M, const float Q[6], double eps,
                 double acc[3], double *phi) {
  Tree t;
  t.cx = {com[0]}; t.cy = {com[1]}; t.cz = {com[2]}; t.cM = {M};
  t.qxx = {Q[0]}; t.qyy = {Q[1]}; t.qzz = {Q[2]}; t.qxy = {Q[3]}; t.qxz = {Q[4]}; t.qyz = {Q[5]};
  acc[0] = acc[1] = acc[2] = 0; *phi = 0;
  eval_pc(t, 0, target[0], target[1], target[2], eps * eps, acc, *phi);
}

void *orc_tree_create(const float *pos, const float *mass, int64_t N, int leaf_size, int group_size, int *err) {
  *err = 0;
  if (!pos || !mass || N <= 0 || N > 2147483647LL || leaf_size < 1 || group_size < 1) { *err = -1; return nullptr; }
  Tree *t = new Tree();
  t->N = N; t->leaf_size = leaf_size; t->group_size = group_size;
  t->pos.assign(pos, pos + 3 * N);
  t->mass.assign(mass, mass + N);
  int rc = build(*t);
  if (rc != 0) { *err = rc; delete t; return nullptr; }
  return t;
}
void orc_tree_destroy(void *h) { delete (Tree *)h; }

int64_t orc_tree_n_cells(void *h) { return (int64_t)((Tree *)h)->cells.size(); }
int64_t orc_tree_n_groups(void *h) { return ((Tree *)h)->n_groups(); }

void orc_tree_get_grid(void *h, float lo[3], float hi[3], float origin[3], int *k) {
  Tree *t = (Tree *)h;
  for (int d = 0; d < 3; ++d) { lo[d] = t->lo[d]; hi[d] = t->hi[d]; origin[d] = t->origin[d]; }
  *k = t->k;
}
void orc_tree_get_keys(void *h, uint64_t *key_caller_order, uint32_t *order, uint64_t *sorted_key) {
  Tree *t = (Tree *)h;
  if (key_caller_order) std::memcpy(key_caller_order, t->key.data(), t->N * sizeof(uint64_t));
  if (order) std::memcpy(order, t->order.data(), t->N * sizeof(uint32_t));
  if (sorted_key) std::memcpy(sorted_key, t->skey.data(), t->N * sizeof(uint64_t));
}
// cells: int32 [n_cells][5] = level, first, count, first_child (-1 leaf), n_child
void orc_tree_get_cells(void *h, int32_t *out) {
  Tree *t = (Tree *)h;
  for (size_t c = 0; c < t->cells.size(); ++c) {
    const Cell &cl = t->cells[c];
    out[5 * c] = cl.level; out[5 * c + 1] = (int32_t)cl.first; out[5 * c + 2] = (int32_t)cl.count;
    out[5 * c + 3] = cl.first_child; out[5 * c + 4] = cl.n_child;
  }
}
// moments: float [n_cells][11] = M, cx, cy, cz, Qxx, Qyy, Qzz, Qxy, Qxz, Qyz, delta
void orc_tree_get_moments(void *h, float *out) {
  Tree *t = (Tree *)h;
  for (size_t c = 0; c < t->cells.size(); ++c) {
    float *o = out + 11 * c;
    o[0] = t->cM[c]; o[1] = t->cx[c]; o[2] = t->cy[c]; o[3] = t->cz[c];
    o[4] = t->qxx[c]; o[5] = t->qyy[c]; o[6] = t->qzz[c]; o[7] = t->qxy[c]; o[8] = t->qxz[c]; o[9] = t->qyz[c];
    o[10] = t->delta[c];
  }
}
// Override the stored FP32 moments (used only if the CUDA path chooses another summation scheme,
// so that walk and forces are compared "on the same tree", north_star).
void orc_tree_set_moments(void *h, const float *in) {
  Tree *t = (Tree *)h;
  for (size_t c = 0; c < t->cells.size(); ++c) {
    const float *o = in + 11 * c;
    t->cM[c] = o[0]; t->cx[c] = o[1]; t->cy[c] = o[2]; t->cz[c] = o[3];
    t->qxx[c] = o[4]; t->qyy[c] = o[5]; t->qzz[c] = o[6]; t->qxy[c] = o[7]; t->qxz[c] = o[8]; t->qyz[c] = o[9];
    t->delta[c] = o[10];
  }
}
void orc_tree_get_groups(void *h, float *gmin, float *gmax) {
  Tree *t = (Tree *)h;
  std::memcpy(gmin, t->gmin.data(), t->gmin.size() * sizeof(float));
  std::memcpy(gmax, t->gmax.data(), t->gmax.size() * sizeof(float));
}
void orc_tree_get_sorted(void *h, float *xyzm /*[N][4]*/) {
  Tree *t = (Tree *)h;
  for (int64_t s = 0; s < t->N; ++s) {
    xyzm[4 * s] = t->sx[s]; xyzm[4 * s + 1] = t->sy[s]; xyzm[4 * s + 2] = t->sz[s]; xyzm[4 * s + 3] = t->sm[s];
  }
}

// T9-T11 for groups g0, g0+stride, ...; acc [N][3] / pot [N] FP64 in original order (entries of
// particles in groups not visited are left untouched). Counts per group via orc_tree_get_counts.
int orc_tree_force(void *h, float theta, float eps, double *acc, double *pot, int64_t g0, int64_t stride) {
  Tree *t = (Tree *)h;
  if (!t || !(theta >= 0.0f) || !(eps >= 0.0f) || g0 < 0 || stride < 1) return -1;
  tree_force(*t, theta, eps, acc, pot, g0, stride);
  return 0;
}
void orc_tree_get_counts(void *h, uint32_t *npp, uint32_t *npc) {
  Tree *t = (Tree *)h;
  std::memcpy(npp, t->npp.data(), t->npp.size() * sizeof(uint32_t));
  std::memcpy(npc, t->npc.data(), t->npc.size() * sizeof(uint32_t));
}
// option "relative": amag = |a| of every particle (caller order, FP32: an input, e.g. of an earlier force pass);
// the scale of group g is alpha * min over its particles (one FP32 multiplication)
int orc_tree_set_mac_relative(void *h, float alpha, const float *amag) {
  Tree *t = (Tree *)h;
  if (!(alpha >= 0.0f) || !amag) return -1;
  const int64_t ng = t->n_groups();
  t->gscale.assign(ng, 0.0f);
  for (int64_t g = 0; g < ng; ++g) {
    const int64_t a0 = g * t->group_size, b0 = std::min<int64_t>(a0 + t->group_size, t->N);
    float m = amag[t->order[a0]];
    for (int64_t s = a0 + 1; s < b0; ++s) m = std::min(m, amag[t->order[s]]);
    t->gscale[g] = alpha * m;
  }
  t->mac = 2;
  return 0;
}
// option "bmax": kind 0 = canonical (S5), 1 = bmax
int orc_tree_set_mac(void *h, int kind) {
  if (kind != 0 && kind != 1) return -1;
  ((Tree *)h)->mac = kind;
  return 0;
}

// [n_cells][7]: tight box lo x,y,z, hi x,y,z, bounding radius b
void orc_tree_get_tight(void *h, float *out) {
  Tree *t = (Tree *)h;
  for (size_t c = 0; c < t->cells.size(); ++c) {
    for (int d = 0; d < 3; ++d) { out[7 * c + d] = t->tlo[3 * c + d]; out[7 * c + 3 + d] = t->thi[3 * c + d]; }
    out[7 * c + 6] = t->brad[c];
  }
}

void orc_tree_get_ropen2(void *h, float *out) {
  Tree *t = (Tree *)h;
  std::memcpy(out, t->ropen2.data(), t->ropen2.size() * sizeof(float));
}
// Diagnostic for the tolerance statement of the force parity: for the particles in the given sorted
// SLOTS, A_i = sum over the interaction list of the MAGNITUDES |a_ij| of the terms whose vector sum is a_i (each term
// evaluated by eval_pp / eval_pc alone).  A_i / |a_i| is the cancellation factor of the sum.  Adds nothing to T1-T12.
int orc_tree_abs_sum(void *h, float theta, float eps, const int64_t *slots, int64_t n, double *out) {
  Tree *t = (Tree *)h;
  if (!t || !slots || !out || !(theta >= 0.0f) || !(eps >= 0.0f)) return -1;
  set_opening(*t, theta);
  const double eps2 = (double)eps * (double)eps;
  for (int64_t k = 0; k < n; ++k) {
    const int64_t s = slots[k];
    if (s < 0 || s >= t->N) return -1;
    std::vector<int32_t> ac, ol;
    walk_group(*t, s / t->group_size, ac, ol);
    const double tx = t->sx[s], ty = t->sy[s], tz = t->sz[s];
    double A = 0.0;
    for (int32_t c : ol) {
      const Cell &cl = t->cells[c];
      for (uint32_t p = cl.first; p < cl.first + cl.count; ++p) {
        if ((int64_t)p == s) continue;
        double a[3] = {0, 0, 0}, phi = 0;
        eval_pp(tx, ty, tz, t->sx[p], t->sy[p], t->sz[p], t->sm[p], eps2, a, phi);
        A += std::sqrt(a[0] * a[0] + a[1] * a[1] + a[2] * a[2]);
      }
    }
    for (int32_t c : ac) {
      double a[3] = {0, 0, 0}, phi = 0;
      eval_pc(*t, c, tx, ty, tz, eps2, a, phi);
      A += std::sqrt(a[0] * a[0] + a[1] * a[1] + a[2] * a[2]);
    }
    out[k] = A;
  }
  return 0;
}

// Interaction lists of one group for the last theta set by orc_tree_force / this call (T10).
// Returns counts through n_acc / n_open; arrays must hold n_cells entries each.
int orc_tree_walk_lists(void *h, float theta, int64_t g, int32_t *acc_cells, int64_t *n_acc,
                        int32_t *open_leaves, int64_t *n_open) {
  Tree *t = (Tree *)h;
  if (g < 0 || g >= t->n_groups()) return -1;
  set_opening(*t, theta);
  std::vector<int32_t> ac, ol;
  walk_group(*t, g, ac, ol);
  std::copy(ac.begin(), ac.end(), acc_cells); *n_acc = (int64_t)ac.size();
  std::copy(ol.begin(), ol.end(), open_leaves); *n_open = (int64_t)ol.size();
  return 0;
}

// T12: nsteps of kick-drift-kick with the tree force. FP32 state, fmaf.
// pos/vel [N][3] updated in place; acc_io [N][3] + pot_io [N] FP32: on entry the force at pos
// (if have_force != 0), on exit the force at the final pos. energies [nsteps+1][2] = kinetic,
// potential (= 1/2 sum m phi) at the start and after every step (FP64 sums, original order).
int orc_leapfrog(float *pos, float *vel, const float *mass, int64_t N, float dt, int nsteps,
                 float theta, float eps, int leaf_size, int group_size,
                 float *acc_io, float *pot_io, int have_force, double *energies) {
  if (!pos || !vel || !mass || N <= 0 || !acc_io || !pot_io) return -1;
  std::vector<double> a(3 * N), p(N);
  auto force = [&]() -> int {
    int err = 0;
    Tree *t = (Tree *)orc_tree_create(pos, mass, N, leaf_size, group_size, &err);
    if (!t) return err;
    tree_force(*t, theta, eps, a.data(), p.data(), 0, 1);
    delete t;
    for (int64_t i = 0; i < 3 * N; ++i) acc_io[i] = (float)a[i];
    for (int64_t i = 0; i < N; ++i) pot_io[i] = (float)p[i];
    return 0;
  };
  auto energy = [&](double *e) {
    double ke = 0, pe = 0;
    for (int64_t i = 0; i < N; ++i) {
      double vx = vel[3 * i], vy = vel[3 * i + 1], vz = vel[3 * i + 2];
      ke += 0.5 * (double)mass[i] * (vx * vx + vy * vy + vz * vz);
      pe += 0.5 * (double)mass[i] * (double)pot_io[i];
    }
    e[0] = ke; e[1] = pe;
  };
  if (!have_force) { int rc = force(); if (rc) return rc; }
  if (energies) energy(energies);
  const float hdt = 0.5f * dt;
  for (int s = 0; s < nsteps; ++s) {
    for (int64_t i = 0; i < 3 * N; ++i) {
      vel[i] = std::fmaf(acc_io[i], hdt, vel[i]);
      pos[i] = std::fmaf(vel[i], dt, pos[i]);
    }
    int rc = force();
    if (rc) return rc;
    for (int64_t i = 0; i < 3 * N; ++i) vel[i] = std::fmaf(acc_io[i], hdt, vel[i]);
    if (energies) energy(energies + 2 * (s + 1));
  }
  return 0;
}

}  // extern "C"
