// Shared device code of the force pass (sm_100a): the per-warp shared-memory block, the p-p / p-c evaluators (scalar and
// packed FP32x2), the compensated running totals and the staging of sources.  Included by bh_force.cu (the fused walk +
// force kernel) and by bh_measure.cu (the measurement aid that runs walk and evaluation as two kernels).
#pragma once
#include <algorithm>
#include <cmath>

#include "bh_common.cuh"

namespace bh {

// Inclusive scan over the warp.  shfl.up reports through its predicate whether the source lane exists, so each
// step is SHFL + predicated IADD (the portable form needs a lane compare and a select per step as well).
__device__ __forceinline__ unsigned warp_incl_scan_u(unsigned v, int /*lane*/) {
#pragma unroll
  for (int o = 1; o < 32; o <<= 1)
    asm volatile("{ .reg .pred p; .reg .b32 r; shfl.sync.up.b32 r|p, %0, %1, 0, 0xffffffff; @p add.u32 %0, %0, r; }"
                 : "+r"(v)
                 : "r"(o));
  return v;
}

// ------------------------------------------------------------------------------------------
// a9 + a10: fused walk + force. One warp per group of 32*TPL consecutive slots.
//
// Walk: a per-warp stack of child RANGES (first_cell << 3 | n-1) in shared memory. Each step pops
// exactly min(32, cells on the stack) cells (splitting the straddling range), tests one cell per
// lane against the group's AABB, and by ballot/prefix compaction appends accepted cells to the
// p-c queue, opened leaves (as particle ranges) to the p-p queue and the child ranges of opened
// internal cells to the stack (deeper ranges on top, so each level holds at most 32 ranges and
// the stack never exceeds 32 * 22 entries: DESIGN.md §Walk).
// Evaluate: whenever a queue holds >= 32 sources, 32 of them are staged in shared memory as float4
// and every lane evaluates them against its TPL targets with broadcast LDS.128 loads.
// ------------------------------------------------------------------------------------------
// sources per unrolled evaluator loop body.  p-c: the whole tile (32 x 32 packed instructions, no loop): 970.8 ms against 976.2 ms with
// 16 at N = 134 M, 55.36 / 55.56 ms at 8.4 M; p-p stays at 16 (32 for both: 1015 ms, the two bodies no longer fit the instruction cache).
// With the relative criterion the lists are half as long and the kernel changes between walking and evaluating twice as often: there
// the 19 KB tile costs more than it gains (459.5 against 453.6 ms per step at 134 M), so those kernels keep 16.
constexpr int PP_UNROLL = 16, PC_UNROLL = 32, PC_UNROLL_REL = 16;
constexpr int WALK_WARPS = 4;  // warps per block of the walk kernels
constexpr int WALK_MINB = 5;  // resident blocks per SM the register budget is sized for
// four targets per lane (group 128) keep twice the per-target state in registers: fewer, fatter blocks
constexpr int walk_minb(int tpl) { return tpl >= 4 ? 3 : WALK_MINB; }
constexpr int COUNT_MINB = 8;            // same for the counting pre-pass (38 registers; shared memory allows 8 blocks)
constexpr unsigned COUNT_TRUNC = 1024;  // the counting walk treats cells this small as opened leaves
constexpr int FOLD_EVERY = 2;  // tiles (of 32 sources) summed in plain FP32 between compensated folds
constexpr int DEFER_CAP = 256;   // deferred child ranges one part of a split group may own
constexpr int STACK_CAP = 1024;  // >= 32 per level (depth-first: 32 x 22) + DEFER_CAP

struct __align__(16) WarpSmem {
  float4 pc0[32], pc1[32], pc2[32];  // cx,cy,cz,M | 2.5 Q'xx,Q'yy,Q'zz, 2.5 tr(Q) eps^2 | 2.5 Q'xy,Q'xz,Q'yz (pc_one)
  float4 pp[32];                     // x,y,z,m
  uint32_t ppidx[32];                // slot of each staged p-p source (self-skip by index, S2)
  uint2 ppq[64];                     // pending particle ranges (first, count)
  uint32_t pcq[64];                  // pending accepted cells
  uint32_t stack[STACK_CAP];
};

struct WalkParams {
  const float4 *spos;
  const float4 *c_test;
  const uint2 *c_link;
  const float4 *c_cm, *c_qa, *c_qb;
  const float *gbox;
  float4 *sacc;            // this context's result buffer of the current pass
  uint2 *gcount;           // this context's per-group counts of the current pass
  float4 *peer_sacc[TREE_SHARD_MAX_WORLD];   // sharded pass: the same two buffers of every attached context
  uint2 *peer_gcount[TREE_SHARD_MAX_WORLD];  // (peer stores over NVLink); n_peers = 0 otherwise
  int n_peers;
  DevInfo *info;
  const uint32_t *c_count; // particles per cell (counting walk only)
  const uint32_t *tasks;   // task = group | part << TASK_GROUP_BITS
  const uint8_t *gparts;   // parts per group (1 = not split)
  uint32_t *gdone;         // finished parts per split group
  float4 *part;            // partial sums of split groups, [task][group size]
  const uint32_t *gthresh; // split groups: cells with at most this many particles are dealt out, not expanded, in the prefix
  uint4 *trace;            // per task: start ns (lo 32), duration ns, SM id, task word (tracing aid)
  long long N;
  unsigned n_groups;
  float eps2;
  float4 *svel;            // tree_leapfrog on one context: the step's closing half kick, v += a * kick_hdt, is applied here in
  float kick_hdt;          // the epilogue (nullptr otherwise: a sharded pass kicks after its barrier)
  int reuse_mode;          // 0: costs from the counting walk; 1: from the previous pass's counts; 2: info->reuse_costs decides
  const uint32_t *order;   // tree_force with caller arrays on one context: the epilogue also writes each result to the caller's
  float *out_acc, *out_pot;  // arrays at order[slot] (a11 fused: no separate pass); order = nullptr otherwise
  const float *c_q;        // relative criterion (walk kernels with REL = true): M l^3 per cell,
  const float *gscale;     // alpha * min |a| per group
};

constexpr unsigned TASK_GROUP_BITS = 26;
constexpr unsigned TASK_GROUP_MASK = (1u << TASK_GROUP_BITS) - 1u;
constexpr unsigned TASK_NONE = 0xffffffffu;  // hole in the task list
constexpr unsigned PARTS_MASK = 0x7fu;       // gparts: number of parts | PARTS_HEAD for expensive groups
constexpr unsigned PARTS_HEAD = 0x80u;

template <int TPL>
struct Targets {
  float x[TPL], y[TPL], z[TPL];
  float ax[TPL], ay[TPL], az[TPL], ph[TPL];  // sums over the tiles evaluated since the last fold
  float phq[TPL];                            // quadrupole part of the potential, scaled (see pc_one)
  uint32_t slot[TPL];
  unsigned long long xp, yp, zp;             // two targets per lane, packed evaluators: x, y, z as FP32x2 register pairs
};

// Running totals (S14).  The per-lane FP32 sums over the last FOLD_EVERY tiles are folded into totals that
// do not drift with the list length: unevaluated FP32 (hi, lo) pairs updated by an error-free two-sum (7 FADD per value).
// BH_PACKED = 0 builds the scalar evaluators for group size 64 too (tests/test_gpu_variants.py compares the two forms
// byte for byte); FP32x2 register pairs: see "Packed evaluators" below.
#ifndef BH_PACKED
#define BH_PACKED 1
#endif
typedef unsigned long long f32x2;  // (lo = target 0, hi = target 1)
__device__ __forceinline__ f32x2 pk2(float lo, float hi) { f32x2 r; asm("mov.b64 %0, {%1,%2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ f32x2 bc2(float s) { return pk2(s, s); }
__device__ __forceinline__ void up2(f32x2 v, float &lo, float &hi) { asm("mov.b64 {%0,%1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b) { f32x2 r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ f32x2 sub2(f32x2 a, f32x2 b) { f32x2 r; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) { f32x2 r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) { f32x2 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }


__device__ __forceinline__ void two_sum_fold(float &hi, float &lo, float x) {
  float s = __fadd_rn(hi, x);
  float bb = __fsub_rn(s, hi);
  float e = __fadd_rn(__fsub_rn(hi, __fsub_rn(s, bb)), __fsub_rn(x, bb));
  hi = s;
  lo = __fadd_rn(lo, e);
}

template <int TPL>
struct Totals {
  float hi[4][TPL], lo[4][TPL];
  __device__ __forceinline__ void clear() {
#pragma unroll
    for (int t = 0; t < TPL; ++t)
#pragma unroll
      for (int c = 0; c < 4; ++c) { hi[c][t] = 0.0f; lo[c][t] = 0.0f; }
  }
  __device__ __forceinline__ void add(int c, int t, float x) { two_sum_fold(hi[c][t], lo[c][t], x); }
  // the potential is a sum of terms of one sign (the quadrupole part is a small correction): no cancellation, so a
  // plain FP32 total over the folds (one rounding per fold, random sign) stays below 1e-6 relative
  __device__ __forceinline__ void add_same_sign(int t, float x) { hi[3][t] = __fadd_rn(hi[3][t], x); }
  __device__ __forceinline__ float get(int c, int t) const { return __fadd_rn(hi[c][t], lo[c][t]); }
};

template <int TPL>
__device__ __forceinline__ void fold_tile(Targets<TPL> &T, Totals<TPL> &R) {
#if BH_PACKED
  if constexpr (TPL == 2) {  // the same two-sums on register pairs: both targets per instruction
    float *const comp[3] = {T.ax, T.ay, T.az};
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const f32x2 hi = pk2(R.hi[c][0], R.hi[c][1]), x = pk2(comp[c][0], comp[c][1]);
      const f32x2 s = add2(hi, x);
      const f32x2 bb = sub2(s, hi);
      const f32x2 e = add2(sub2(hi, sub2(s, bb)), sub2(x, bb));
      const f32x2 lo = add2(pk2(R.lo[c][0], R.lo[c][1]), e);
      up2(s, R.hi[c][0], R.hi[c][1]);
      up2(lo, R.lo[c][0], R.lo[c][1]);
    }
    // (keeping the low words in shared memory instead frees 6 registers but ran 2.5 % slower)
#pragma unroll
    for (int t = 0; t < 2; ++t) {
      R.add_same_sign(t, fmaf(-0.2f, T.phq[t], T.ph[t]));
      T.ax[t] = T.ay[t] = T.az[t] = T.ph[t] = T.phq[t] = 0.0f;
    }
    return;
  }
#endif
#pragma unroll
  for (int t = 0; t < TPL; ++t) {
    R.add(0, t, T.ax[t]);
    R.add(1, t, T.ay[t]);
    R.add(2, t, T.az[t]);
    R.add_same_sign(t, fmaf(-0.2f, T.phq[t], T.ph[t]));
    T.ax[t] = T.ay[t] = T.az[t] = T.ph[t] = T.phq[t] = 0.0f;
  }
}

// MUFU.RSQ without the denormal range fix-up of rsqrtf(): the argument is r^2 + eps^2 of FP32
// coordinates, never subnormal unless the particles coincide with eps = 0 (excluded by the ABI).
__device__ __forceinline__ float rsqrt_fast(float x) {
  float y;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

template <int TPL, bool MASK>
__device__ __forceinline__ void pp_one(const float4 s, uint32_t sidx, Targets<TPL> &T, float eps2) {
#pragma unroll
  for (int t = 0; t < TPL; ++t) {
    float dx = s.x - T.x[t], dy = s.y - T.y[t], dz = s.z - T.z[t];
    float r2 = fmaf(dx, dx, eps2);
    r2 = fmaf(dy, dy, r2);
    r2 = fmaf(dz, dz, r2);
    float m = s.w;
    if (MASK) {
      if (sidx == T.slot[t]) { m = 0.0f; r2 = 1.0f; }
    }
    float ri = rsqrt_fast(r2);
    float ri2 = ri * ri;
    float mr = m * ri;
    float mr3 = mr * ri2;
    T.ax[t] = fmaf(mr3, dx, T.ax[t]);
    T.ay[t] = fmaf(mr3, dy, T.ay[t]);
    T.az[t] = fmaf(mr3, dz, T.az[t]);
    T.ph[t] -= mr;
  }
}

// Particle-cell interaction, Eqs. (1),(2) with s^2 = |r|^2 + eps^2 in every power (S1),
// rearranged exactly: with Q' = 3Q - tr(Q) I and w = r^T Q' r - tr(Q) eps^2,
//   phi = -M rho - 1/2 w rho^5,   a = (M rho^3 + 5/2 w rho^7) r - rho^5 Q' r.
// Staged per source: a = (cx,cy,cz,M), b = 2.5 (Q'xx,Q'yy,Q'zz, tr(Q) eps^2), c = 2.5 (Q'xy,Q'xz,Q'yz).
// The two parts of a are summed separately within a tile, sum g r and sum rho^5 (2.5 Q' r), and joined with the factor
// -0.4 once per tile: 32 FP32 instructions + 1 MUFU per target (the paper counts 65 flop for this interaction).
template <int TPL>
struct QuadAcc {  // sum over one tile of rho^5 (2.5 Q' r) per target; a += -0.4 x that, once per tile (pc_tile_end)
  float x[TPL], y[TPL], z[TPL];
  __device__ __forceinline__ QuadAcc() {
#pragma unroll
    for (int t = 0; t < TPL; ++t) x[t] = y[t] = z[t] = 0.0f;
  }
};

template <int TPL>
__device__ __forceinline__ void pc_one(const float4 a, const float4 b, const float4 c, Targets<TPL> &T, QuadAcc<TPL> &A,
                                       float eps2) {
#pragma unroll
  for (int t = 0; t < TPL; ++t) {
    float dx = a.x - T.x[t], dy = a.y - T.y[t], dz = a.z - T.z[t];
    float r2 = fmaf(dx, dx, eps2);
    r2 = fmaf(dy, dy, r2);
    r2 = fmaf(dz, dz, r2);
    float ri = rsqrt_fast(r2);
    float vx = fmaf(c.y, dz, fmaf(c.x, dy, b.x * dx));   // 2.5 Q' r
    float vy = fmaf(c.z, dz, fmaf(b.y, dy, c.x * dx));
    float vz = fmaf(b.z, dz, fmaf(c.z, dy, c.y * dx));
    float w = fmaf(dz, vz, fmaf(dy, vy, fmaf(dx, vx, -b.w)));  // 2.5 w
    float ri2 = ri * ri;
    float ri3 = ri * ri2;
    float ri4 = ri2 * ri2;
    float ri5 = ri3 * ri2;
    T.ph[t] = fmaf(-a.w, ri, T.ph[t]);       // -M rho
    T.phq[t] = fmaf(w, ri5, T.phq[t]);       // 2.5 w rho^5; folded in as -0.2 x
    float g = fmaf(w, ri4, a.w) * ri3;       // M rho^3 + 2.5 w rho^7
    T.ax[t] = fmaf(g, dx, T.ax[t]);
    T.ay[t] = fmaf(g, dy, T.ay[t]);
    T.az[t] = fmaf(g, dz, T.az[t]);
    A.x[t] = fmaf(ri5, vx, A.x[t]);          // rho^5 (2.5 Q' r): - rho^5 Q' r = -0.4 x this, applied per tile
    A.y[t] = fmaf(ri5, vy, A.y[t]);
    A.z[t] = fmaf(ri5, vz, A.z[t]);
  }
}

template <int TPL>
__device__ __forceinline__ void pc_tile_end(Targets<TPL> &T, const QuadAcc<TPL> &A) {
#pragma unroll
  for (int t = 0; t < TPL; ++t) {
    T.ax[t] = fmaf(-0.4f, A.x[t], T.ax[t]);
    T.ay[t] = fmaf(-0.4f, A.y[t], T.ay[t]);
    T.az[t] = fmaf(-0.4f, A.z[t], T.az[t]);
  }
}

// ------------------------------------------------------------------------------------------
// Packed evaluators for two targets per lane (group size 64): sm_100a has FP32x2 instructions (FADD2 / FMUL2 /
// FFMA2) that work on aligned register pairs and take a scalar register as a broadcast operand, so one instruction
// serves both targets of a lane with the source operand read once.  Same operations in the same order as pp_one /
// pc_one, each IEEE round-to-nearest: the results are bit-identical.  The pair operands are always spread over both
// register-file banks, which is what the scalar form cannot arrange:
// in isolation the p-c loop runs at 0.77 of the FP32 peak against 0.69 (micro-benchmark), with half the instructions.
// ------------------------------------------------------------------------------------------
struct Targets2 {  // the packed view of Targets<2> during one tile
  f32x2 x, y, z, ax, ay, az, ph, phq;
  f32x2 qx = 0ull, qy = 0ull, qz = 0ull;  // p-c tiles: sum of rho^5 (2.5 Q' r) over the tile (pc_tile_end2)
  __device__ __forceinline__ explicit Targets2(const Targets<2> &T)
      :
        x(T.xp), y(T.yp), z(T.zp),  // packed once when the task loads its targets (walk_task)
        ax(pk2(T.ax[0], T.ax[1])),
        ay(pk2(T.ay[0], T.ay[1])), az(pk2(T.az[0], T.az[1])), ph(pk2(T.ph[0], T.ph[1])), phq(pk2(T.phq[0], T.phq[1])) {}
  __device__ __forceinline__ void pc_tile_end2() {  // a += -0.4 x the tile's sum of rho^5 (2.5 Q' r)
    const f32x2 m = bc2(-0.4f);
    ax = fma2(m, qx, ax); ay = fma2(m, qy, ay); az = fma2(m, qz, az);
  }
  __device__ __forceinline__ void store(Targets<2> &T) const {
    up2(ax, T.ax[0], T.ax[1]); up2(ay, T.ay[0], T.ay[1]); up2(az, T.az[0], T.az[1]);
    up2(ph, T.ph[0], T.ph[1]); up2(phq, T.phq[0], T.phq[1]);
  }
};

template <bool MASK>
__device__ __forceinline__ void pp_one2(const float4 s, uint32_t sidx, const uint32_t (&slot)[2], Targets2 &T, f32x2 eps2) {
  const f32x2 dx = sub2(bc2(s.x), T.x), dy = sub2(bc2(s.y), T.y), dz = sub2(bc2(s.z), T.z);
  f32x2 r2 = fma2(dx, dx, eps2);
  r2 = fma2(dy, dy, r2);
  r2 = fma2(dz, dz, r2);
  float r2a, r2b, m0 = s.w, m1 = s.w;
  up2(r2, r2a, r2b);
  if (MASK) {
    if (sidx == slot[0]) { m0 = 0.0f; r2a = 1.0f; }
    if (sidx == slot[1]) { m1 = 0.0f; r2b = 1.0f; }
  }
  const f32x2 ri = pk2(rsqrt_fast(r2a), rsqrt_fast(r2b));
  const f32x2 ri2 = mul2(ri, ri);
  const f32x2 mr = mul2(MASK ? pk2(m0, m1) : bc2(s.w), ri);
  const f32x2 mr3 = mul2(mr, ri2);
  T.ax = fma2(mr3, dx, T.ax);
  T.ay = fma2(mr3, dy, T.ay);
  T.az = fma2(mr3, dz, T.az);
  T.ph = sub2(T.ph, mr);
}

// see pc_one for the formulas; a = (cx,cy,cz,M), b = 2.5 (Q'xx,Q'yy,Q'zz, tr(Q) eps^2), c = 2.5 (Q'xy,Q'xz,Q'yz)
__device__ __forceinline__ void pc_one2(const float4 a, const float4 b, const float4 c, Targets2 &T, f32x2 eps2) {
  const f32x2 dx = sub2(bc2(a.x), T.x), dy = sub2(bc2(a.y), T.y), dz = sub2(bc2(a.z), T.z);
  f32x2 r2 = fma2(dx, dx, eps2);
  r2 = fma2(dy, dy, r2);
  r2 = fma2(dz, dz, r2);
  float r2a, r2b;
  up2(r2, r2a, r2b);
  const f32x2 ri = pk2(rsqrt_fast(r2a), rsqrt_fast(r2b));
  const f32x2 vx = fma2(bc2(c.y), dz, fma2(bc2(c.x), dy, mul2(bc2(b.x), dx)));
  const f32x2 vy = fma2(bc2(c.z), dz, fma2(bc2(b.y), dy, mul2(bc2(c.x), dx)));
  const f32x2 vz = fma2(bc2(b.z), dz, fma2(bc2(c.z), dy, mul2(bc2(c.y), dx)));
  const f32x2 w = fma2(dz, vz, fma2(dy, vy, fma2(dx, vx, bc2(-b.w))));
  const f32x2 ri2 = mul2(ri, ri);
  const f32x2 ri3 = mul2(ri, ri2);
  const f32x2 ri4 = mul2(ri2, ri2);
  const f32x2 ri5 = mul2(ri3, ri2);
  T.ph = fma2(bc2(-a.w), ri, T.ph);
  T.phq = fma2(w, ri5, T.phq);
  const f32x2 g = mul2(fma2(w, ri4, bc2(a.w)), ri3);
  T.ax = fma2(g, dx, T.ax); T.ay = fma2(g, dy, T.ay); T.az = fma2(g, dz, T.az);
  T.qx = fma2(ri5, vx, T.qx); T.qy = fma2(ri5, vy, T.qy); T.qz = fma2(ri5, vz, T.qz);
}

template <int TPL>
__device__ __forceinline__ void eval_pp_tile(const WarpSmem &ws, int cnt, bool mask, Targets<TPL> &T, float eps2) {
  if constexpr (TPL == 2 && BH_PACKED) {
    Targets2 P2(T);
    const f32x2 e2 = bc2(eps2);
    const uint32_t slot[2] = {T.slot[0], T.slot[1]};
    if (!mask && cnt == 32) {
#pragma unroll(PP_UNROLL)
      for (int j = 0; j < 32; ++j) pp_one2<false>(ws.pp[j], 0u, slot, P2, e2);
    } else if (!mask) {
      for (int j = 0; j < cnt; ++j) pp_one2<false>(ws.pp[j], 0u, slot, P2, e2);
    } else {
#pragma unroll 2
      for (int j = 0; j < cnt; ++j) pp_one2<true>(ws.pp[j], ws.ppidx[j], slot, P2, e2);
    }
    P2.store(T);
    return;
  }
  if (!mask && cnt == 32) {
#pragma unroll(PP_UNROLL)
    for (int j = 0; j < 32; ++j) pp_one<TPL, false>(ws.pp[j], 0u, T, eps2);
  } else if (!mask) {
    for (int j = 0; j < cnt; ++j) pp_one<TPL, false>(ws.pp[j], 0u, T, eps2);
  } else {
#pragma unroll 2
    for (int j = 0; j < cnt; ++j) pp_one<TPL, true>(ws.pp[j], ws.ppidx[j], T, eps2);
  }
}

template <int TPL, int PCU = PC_UNROLL>
__device__ __forceinline__ void eval_pc_tile(const WarpSmem &ws, int cnt, Targets<TPL> &T, float eps2) {
  if constexpr (TPL == 2 && BH_PACKED) {
    Targets2 P2(T);
    const f32x2 e2 = bc2(eps2);
    if (cnt == 32) {
#pragma unroll(PCU)
      for (int j = 0; j < 32; ++j) pc_one2(ws.pc0[j], ws.pc1[j], ws.pc2[j], P2, e2);
    } else {
      for (int j = 0; j < cnt; ++j) pc_one2(ws.pc0[j], ws.pc1[j], ws.pc2[j], P2, e2);
    }
    P2.pc_tile_end2();
    P2.store(T);
    return;
  }
  QuadAcc<TPL> A;
  if (cnt == 32) {
#pragma unroll(PCU)
    for (int j = 0; j < 32; ++j) pc_one<TPL>(ws.pc0[j], ws.pc1[j], ws.pc2[j], T, A, eps2);
  } else {
    for (int j = 0; j < cnt; ++j) pc_one<TPL>(ws.pc0[j], ws.pc1[j], ws.pc2[j], T, A, eps2);
  }
  pc_tile_end<TPL>(T, A);
}

// Take `want` (<= 32) particles from the back of the p-p range queue; if `load`, stage them.
// Returns true if any staged source is one of this group's own slots.
__device__ __forceinline__ bool stage_pp(WarpSmem &ws, int lane, int &entries, int want, bool load,
                                         const float4 *__restrict__ spos, uint32_t g0, uint32_t gsize) {
  const bool have = lane < entries;
  uint2 e = have ? ws.ppq[entries - 1 - lane] : make_uint2(0u, 0u);
  const unsigned n = have ? min(e.y, 33u) : 0u;  // clamp: only "more than 32" matters
  const unsigned incl = warp_incl_scan_u(n, lane), excl = incl - n;
  const bool take = have && excl < (unsigned)want;
  const bool full = incl <= (unsigned)want;
  if (take && !full) {
    unsigned k = (unsigned)want - excl;
    ws.ppq[entries - 1 - lane] = make_uint2(e.x + k, e.y - k);
  }
  entries -= __popc(__ballot_sync(0xffffffffu, take && full));
  bool any_own = false;
  if (load) {  // warp-uniform
    const unsigned head = __reduce_or_sync(0xffffffffu, take ? (1u << excl) : 0u);
    const int ei = __popc(head & (0xffffffffu >> (31 - lane))) - 1;
    const unsigned fx = __shfl_sync(0xffffffffu, e.x, ei & 31);
    const unsigned ex = __shfl_sync(0xffffffffu, excl, ei & 31);
    const unsigned pidx = fx + ((unsigned)lane - ex);
    const bool valid = lane < want;
    if (valid) {
      ws.pp[lane] = spos[pidx];
      ws.ppidx[lane] = pidx;
    }
    any_own = __any_sync(0xffffffffu, valid && (pidx - g0) < gsize);
  }
  __syncwarp();
  return any_own;
}

__device__ __forceinline__ void stage_pc(WarpSmem &ws, int lane, int cnt, const WalkParams &P) {
  if (lane < cnt) {
    const unsigned c = ws.pcq[lane];
    const float4 a = P.c_cm[c], qa = P.c_qa[c], qb = P.c_qb[c];
    const float tr = qb.w;
    ws.pc0[lane] = a;
    ws.pc1[lane] = make_float4(2.5f * fmaf(3.0f, qa.x, -tr), 2.5f * fmaf(3.0f, qa.y, -tr), 2.5f * fmaf(3.0f, qa.z, -tr),
                               2.5f * tr * P.eps2);
    ws.pc2[lane] = make_float4(7.5f * qb.x, 7.5f * qb.y, 7.5f * qb.z, 0.0f);
  }
  __syncwarp();
}

}  // namespace bh
