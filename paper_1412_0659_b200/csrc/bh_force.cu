// Force-pass kernels (sm_100a): opening radii, the fused tree-walk + force kernel, un-permute,
// leapfrog and energy.  The walk+force kernel is bound by the FP32 FMA pipe;
// it is not a dense contraction, so no tensor cores (north_star).
#include <algorithm>
#include <cmath>

#include "bh_common.cuh"
#include "bh_eval.cuh"

namespace bh {
// ------------------------------------------------------------------------------------------
// a8: opening radius per cell for this theta, packed with the centre of mass into the 16-byte
// test record (T9): r = l_c / theta; r = r + delta; r_open^2 = r * r, each one IEEE op.
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) opening_kernel(const DevInfo *__restrict__ info, float theta,
                                                      const uint8_t *__restrict__ c_level,
                                                      const float4 *__restrict__ c_cm, const float4 *__restrict__ c_qa,
                                                      const float4 *__restrict__ c_tlo, float4 *__restrict__ c_test,
                                                      float *__restrict__ c_q) {
  long long c = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (info->cells_overflow || c >= info->n_cells) return;
  if (c_q) {  // relative criterion: q = M l^3, three IEEE multiplications in this order
    const float lc = ldexpf(1.0f, info->k - (int)c_level[c]);
    c_q[c] = __fmul_rn(__fmul_rn(__fmul_rn(c_cm[c].w, lc), lc), lc);
  }
  float r;
  if (c_tlo) {  // TREE_MAC_BMAX: r = b / theta (theta = 0 opens everything, also where b = 0)
    r = theta == 0.0f ? INFINITY : __fdiv_rn(c_tlo[c].w, theta);
  } else {
    float lc = ldexpf(1.0f, info->k - (int)c_level[c]);
    r = __fdiv_rn(lc, theta);
    r = __fadd_rn(r, c_qa[c].w);
  }
  float4 cm = c_cm[c];
  c_test[c] = make_float4(cm.x, cm.y, cm.z, __fmul_rn(r, r));
}

// One kernel, two modes.
//  COUNT = true : truncated walk only; writes a cost estimate per group, from which the task list
//                 is built (task kernels below).
//  COUNT = false: work items are TASKS (group g, part j of s). An expensive group is cut into s
//                 parts: all parts repeat a short breadth-first PREFIX of the walk (tiles met
//                 there are dealt out by tile number mod s), then the frontier is dealt out
//                 round-robin (entry i goes to part i mod s) and every part walks and evaluates
//                 its own share depth-first. The parts' partial sums are combined in part order
//                 by the part that finishes last, so the result does not depend on timing.
template <int TPL>
struct WalkState {
  int pp_entries, pp_pending, pc_pending;
  unsigned tile_wait, tile_parts;
  int unfolded;  // tiles accumulated in T since the last fold into the running totals
};

// Evaluate what is left in the two queues as partial tiles (tile ownership by the counter rule).
template <int TPL, int PCU>
__device__ __forceinline__ void flush_queues(WarpSmem &ws, int lane, WalkState<TPL> &S, Targets<TPL> &T, Totals<TPL> &R,
                                             const WalkParams &P, uint32_t g0, uint32_t gsize) {
  if (S.pc_pending > 0) {
    const bool mine = S.tile_wait == 0;
    S.tile_wait = mine ? S.tile_parts - 1 : S.tile_wait - 1;
    if (mine) {
      stage_pc(ws, lane, S.pc_pending, P);
      eval_pc_tile<TPL, PCU>(ws, S.pc_pending, T, P.eps2);
      if (++S.unfolded >= FOLD_EVERY) { fold_tile<TPL>(T, R); S.unfolded = 0; }
      __syncwarp();
    }
    S.pc_pending = 0;
  }
  if (S.pp_pending > 0) {
    const bool mine = S.tile_wait == 0;
    S.tile_wait = mine ? S.tile_parts - 1 : S.tile_wait - 1;
    const bool own = stage_pp(ws, lane, S.pp_entries, S.pp_pending, mine, P.spos, g0, gsize);
    if (mine) {
      eval_pp_tile<TPL>(ws, S.pp_pending, own, T, P.eps2);
      if (++S.unfolded >= FOLD_EVERY) { fold_tile<TPL>(T, R); S.unfolded = 0; }
      __syncwarp();
    }
    S.pp_pending = 0;
    S.pp_entries = 0;
  }
}

// a12, second half kick of a step, fused into the walk's epilogue: v = fma(a, dt/2, v) (T12)
// a11 fused into the epilogue: the result of `slot` to the caller's arrays (caller order).  12- and 4-byte random writes,
// spread over the whole walk (as a pass of their own they ran at a third of the gather's speed).
__device__ __forceinline__ void emit_caller(const WalkParams &P, unsigned slot, const float4 r) {
  const size_t ci = P.order[slot];
  if (P.out_acc) { float *a = P.out_acc + 3 * ci; a[0] = r.x; a[1] = r.y; a[2] = r.z; }
  if (P.out_pot) P.out_pot[ci] = r.w;
}

__device__ __forceinline__ void kick_slot(float4 *v, const float4 a, float hdt) {
  float4 u = *v;
  u.x = __fmaf_rn(a.x, hdt, u.x); u.y = __fmaf_rn(a.y, hdt, u.y); u.z = __fmaf_rn(a.z, hdt, u.z);
  *v = u;
}

// One work item: group g (part `part` of `nparts`).
template <int TPL, bool COUNT, bool REL>
__device__ __forceinline__ void walk_task(const WalkParams &P, WarpSmem &ws, const int lane, const unsigned item,
                                          const unsigned g, const unsigned part, const unsigned nparts,
                                          const unsigned long long t_start) {
  const unsigned lt = (1u << lane) - 1u;
  const unsigned gt = ~((lt << 1) | 1u);
  constexpr unsigned GS = 32u * TPL;
  const bool SPLIT = !COUNT && nparts > 1;
  const long long g0 = (long long)g * GS;
  const long long rem = P.N - g0;
  const unsigned gsize = rem < (long long)GS ? (unsigned)rem : GS;
  Targets<TPL> T;
  Totals<TPL> R;
  R.clear();
#pragma unroll
  for (int t = 0; t < TPL; ++t) {
    unsigned j = lane + 32u * t;
    T.slot[t] = (uint32_t)(g0 + j);
    float4 p = make_float4(0.f, 0.f, 0.f, 0.f);
    if (!COUNT) p = P.spos[g0 + (j < gsize ? j : gsize - 1)];  // padded lanes copy a real target
    T.x[t] = p.x; T.y[t] = p.y; T.z[t] = p.z;
    T.ax[t] = T.ay[t] = T.az[t] = T.ph[t] = T.phq[t] = 0.0f;
    if (j >= gsize) T.slot[t] = 0xffffffffu;
  }
  if constexpr (TPL == 2 && BH_PACKED && !COUNT) {
    // scalar loads: the halves of a pair can then be the load destinations themselves (the quad of an LDG.128 cannot be
    // an aligned pair of two different targets, and ptxas would copy quad -> pair before every use)
    const unsigned j0 = lane < gsize ? lane : gsize - 1, j1 = lane + 32u < gsize ? lane + 32u : gsize - 1;
    const float *a0 = reinterpret_cast<const float *>(P.spos + g0 + j0), *a1 = reinterpret_cast<const float *>(P.spos + g0 + j1);
    float c0[3], c1[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      asm volatile("ld.global.f32 %0, [%1];" : "=f"(c0[c]) : "l"(a0 + c));
      asm volatile("ld.global.f32 %0, [%1];" : "=f"(c1[c]) : "l"(a1 + c));
    }
    T.xp = pk2(c0[0], c1[0]); T.yp = pk2(c0[1], c1[1]); T.zp = pk2(c0[2], c1[2]);
  }
  const float *gb = P.gbox + 6ll * g;
  const float bx0 = gb[0], by0 = gb[1], bz0 = gb[2], bx1 = gb[3], by1 = gb[4], bz1 = gb[5];
  float gscale = 0.0f;  // relative criterion: alpha * min |a| over the group's particles
  if (REL) gscale = P.gscale[g];

  int sp = 1;                       // live stack entries are [0, sp)
  if (lane == 0) ws.stack[0] = 0u;  // root: cell 0, one cell
  __syncwarp();
  WalkState<TPL> S;
  S.pp_entries = 0; S.pp_pending = 0; S.pc_pending = 0;
  S.tile_wait = part; S.tile_parts = nparts; S.unfolded = 0;
  unsigned n_pp = 0, n_pc = 0;
  bool prefix = SPLIT;  // all parts walk the large-cell skeleton identically
  int dp = 0;                          // this part's deferred entries, stored downwards from the end of the stack
  unsigned dcount = 0;                 // deferred entries seen so far by every part (entry i belongs to part i mod s)
  const unsigned small_cell = SPLIT ? P.gthresh[g] : 0u;

  for (;;) {
    // ---- stack empty: evaluate what is left in the queues (the only call site of the partial-tile
    //      evaluators). A part of a split group has then finished the skeleton all parts walk alike and
    //      continues with its own share of the deferred child ranges, evaluating every tile itself.
    if (sp == 0) {
      if (!COUNT) flush_queues<TPL, REL ? PC_UNROLL_REL : PC_UNROLL>(ws, lane, S, T, R, P, (uint32_t)g0, gsize);
      if (!(SPLIT && prefix)) break;
      if constexpr (!COUNT) {
        for (int base = 0; base < dp; base += 32) {
          const int i = base + lane;
          const unsigned e = i < dp ? ws.stack[STACK_CAP - 1 - i] : 0u;
          __syncwarp();
          if (i < dp) ws.stack[i] = e;
        }
        __syncwarp();
        sp = dp; dp = 0;
        prefix = false;
        S.tile_parts = 1; S.tile_wait = 0;
        if (part != 0) { n_pp = 0; n_pc = 0; }  // the prefix is counted by part 0 only
        if (sp == 0) break;
      }
    }
    // ---- pop exactly min(32, cells on stack) cells from the top (deepest first)
    const int live = sp;
    const bool have = lane < live;
    const int my = sp - 1 - lane;
    const unsigned e = have ? ws.stack[my] : 0u;
    const unsigned n = have ? (e & 7u) + 1u : 0u;
    const unsigned incl = warp_incl_scan_u(n, lane), excl = incl - n;
    const bool take = have && excl < 32u;
    const bool full = incl <= 32u;
    if (take && !full) {
      unsigned k = 32u - excl;
      ws.stack[my] = (((e >> 3) + k) << 3) | (n - k - 1u);
    }
    sp -= __popc(__ballot_sync(0xffffffffu, take && full));
    const unsigned tot_all = __shfl_sync(0xffffffffu, incl, 31);
    const unsigned total = tot_all < 32u ? tot_all : 32u;
    const unsigned head = __reduce_or_sync(0xffffffffu, take ? (1u << excl) : 0u);
    const int ei = __popc(head & (0xffffffffu >> (31 - lane))) - 1;
    const unsigned fx = __shfl_sync(0xffffffffu, e >> 3, ei & 31);
    const unsigned ex = __shfl_sync(0xffffffffu, excl, ei & 31);
    const bool valid = (unsigned)lane < total;
    const unsigned cell = fx + ((unsigned)lane - ex);

    // ---- multipole acceptance test (T10), exact op sequence
    bool accept = false, open_leaf = false, open_int = false;
    uint2 lk = make_uint2(0u, 0u);
    if (valid) {
      const float4 tr = P.c_test[cell];
      lk = P.c_link[cell];
      float ux = fmaxf(0.0f, fmaxf(__fsub_rn(bx0, tr.x), __fsub_rn(tr.x, bx1)));
      float uy = fmaxf(0.0f, fmaxf(__fsub_rn(by0, tr.y), __fsub_rn(tr.y, by1)));
      float uz = fmaxf(0.0f, fmaxf(__fsub_rn(bz0, tr.z), __fsub_rn(tr.z, bz1)));
      float d2 = __fmaf_rn(uz, uz, __fmaf_rn(uy, uy, __fmul_rn(ux, ux)));
      accept = d2 > tr.w;
      if (REL) {  // error-targeted condition on top of the geometric floor: D^5 alpha a_g > M l^3, one IEEE op each
        const float lhs = __fmul_rn(__fmul_rn(__fmul_rn(__fsqrt_rn(d2), d2), d2), gscale);
        accept = accept && lhs > P.c_q[cell];
      }
      bool leaf = !(lk.y & LEAF_FLAG);
      if (COUNT && !leaf && !accept) {  // cost estimate: do not descend below small cells
        const unsigned cc = P.c_count[cell];
        if (cc <= COUNT_TRUNC) { leaf = true; lk.y = cc; }
      }
      open_leaf = !accept && leaf;
      open_int = !accept && !leaf;
    }
    // ---- prefix only: an opened cell with few particles is not expanded here; its child range is
    //      entry number dcount of the group's deferred list and belongs to part (dcount mod s)
    if (SPLIT && prefix) {
      const bool small = open_int && P.c_count[cell] <= small_cell;
      const unsigned m = __ballot_sync(0xffffffffu, small);
      if (dcount + __popc(m) <= (unsigned)DEFER_CAP * nparts) {  // the same decision in every part
        const bool mine = small && ((dcount + __popc(m & lt)) % nparts) == part;
        const unsigned mm = __ballot_sync(0xffffffffu, mine);
        if (mine) ws.stack[STACK_CAP - 1 - (dp + __popc(mm & lt))] = (lk.x << 3) | ((lk.y & 0xfu) - 1u);
        if (small) open_int = false;
        dp += __popc(mm);
        dcount += __popc(m);
      }
    }
    // ---- opened internal cells: push child ranges so that the stack stays sorted by level
    //      (prefix: lane order = shallow to deep; afterwards lane 0 holds the deepest cell)
    {
      const unsigned m = __ballot_sync(0xffffffffu, open_int);
      if (open_int) ws.stack[sp + __popc(m & gt)] = (lk.x << 3) | ((lk.y & 0xfu) - 1u);
      sp += __popc(m);
      if (sp + dp + 32 > STACK_CAP) {  // cannot happen within the bounds of DESIGN.md §Walk; never write past the stack
        if (lane == 0) { P.info->walk_overflow = 1u; P.info->walk_overflow_sticky = 1u; }
        sp = 0; dp = 0;
      }
    }
    // ---- accepted cells -> p-c queue
    {
      const unsigned m = __ballot_sync(0xffffffffu, accept);
      if (!COUNT) { if (accept) ws.pcq[S.pc_pending + __popc(m & lt)] = cell; }
      const int c = __popc(m);
      S.pc_pending += c;
      n_pc += c;
    }
    // ---- opened leaves -> p-p range queue
    {
      const unsigned m = __ballot_sync(0xffffffffu, open_leaf);
      if (!COUNT) { if (open_leaf) ws.ppq[S.pp_entries + __popc(m & lt)] = lk; }
      S.pp_entries += __popc(m);
      const unsigned c = __reduce_add_sync(0xffffffffu, open_leaf ? lk.y : 0u);
      S.pp_pending += (int)c;
      n_pp += c;
    }
    __syncwarp();
    if (COUNT) { S.pc_pending = 0; S.pp_pending = 0; S.pp_entries = 0; continue; }
    // ---- evaluate full tiles (only those that belong to this part)
    if (S.pc_pending >= 32) {
      const bool mine = S.tile_wait == 0;
      S.tile_wait = mine ? S.tile_parts - 1 : S.tile_wait - 1;
      if (mine) {
        stage_pc(ws, lane, 32, P);
        eval_pc_tile<TPL, REL ? PC_UNROLL_REL : PC_UNROLL>(ws, 32, T, P.eps2);
        if (++S.unfolded >= FOLD_EVERY) { fold_tile<TPL>(T, R); S.unfolded = 0; }
        __syncwarp();
      }
      // (a ring buffer instead of this shift costs a register: the kernel then spills and runs 1.6 % slower)
      const unsigned mv = (lane + 32 < S.pc_pending) ? ws.pcq[lane + 32] : 0u;
      __syncwarp();
      ws.pcq[lane] = mv;
      S.pc_pending -= 32;
      __syncwarp();
    }
    while (S.pp_pending >= 32) {
      const bool mine = S.tile_wait == 0;
      S.tile_wait = mine ? S.tile_parts - 1 : S.tile_wait - 1;
      const bool own = stage_pp(ws, lane, S.pp_entries, 32, mine, P.spos, (uint32_t)g0, gsize);
      if (mine) {
        eval_pp_tile<TPL>(ws, 32, own, T, P.eps2);
        if (++S.unfolded >= FOLD_EVERY) { fold_tile<TPL>(T, R); S.unfolded = 0; }
      }
      S.pp_pending -= 32;
      __syncwarp();
    }
  }
  if (COUNT) {
    if (lane == 0) {
      const unsigned long long c = 13ull * n_pp + 37ull * n_pc;
      P.gdone[g] = c > 0xffffffffull ? 0xffffffffu : (unsigned)c;  // read and cleared by task_cost_kernel
      atomicAdd(&P.info->sched_cost, c);
    }
    return;
  }
  fold_tile<TPL>(T, R);
  if (prefix && part != 0) { n_pp = 0; n_pc = 0; }  // walk ended inside the prefix: counted by part 0
  if (lane == 0) {
    unsigned long long t_end;
    unsigned smid;
    asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t_end));
    asm volatile("mov.u32 %0, %smid;" : "=r"(smid));
    const unsigned dur = (unsigned)(t_end - t_start);
    if (nparts == 1) {
      P.gcount[g] = make_uint2(n_pp, n_pc);
      for (int q = 0; q < P.n_peers; ++q) P.peer_gcount[q][g] = make_uint2(n_pp, n_pc);
    } else {  // gcount of split groups is zeroed by task_class_kernel
      atomicAdd(&P.gcount[g].x, n_pp);
      atomicAdd(&P.gcount[g].y, n_pc);
    }
    atomicAdd(&P.info->n_pp, (unsigned long long)n_pp * gsize);
    atomicAdd(&P.info->n_pc, (unsigned long long)n_pc * gsize);
    P.trace[item] = make_uint4((unsigned)(t_start - P.info->t0_ns), dur, smid, P.tasks[item]);
  }
  // ---- results
  float4 res[TPL];
#pragma unroll
  for (int t = 0; t < TPL; ++t)
    res[t] = make_float4(R.get(0, t), R.get(1, t), R.get(2, t), R.get(3, t));
  if (nparts == 1) {
#pragma unroll
    for (int t = 0; t < TPL; ++t) {
      unsigned j = lane + 32u * t;
      if (j < gsize) {
        P.sacc[g0 + j] = res[t];
        for (int q = 0; q < P.n_peers; ++q) P.peer_sacc[q][g0 + j] = res[t];
        if (P.svel) kick_slot(P.svel + g0 + j, res[t], P.kick_hdt);
        if (P.order) emit_caller(P, g0 + j, res[t]);
      }
    }
  } else {
    // split group: its parts are consecutive tasks, in the head (expensive groups) or the tail
    // region of the task list; both regions map onto the partial-sum buffer
    const unsigned na = P.info->n_tasks_a;
    const size_t slot = item < na ? item : na + (item - P.info->tail_start);
    float4 *mine = P.part + slot * GS;
#pragma unroll
    for (int t = 0; t < TPL; ++t) __stcg(&mine[lane + 32u * t], res[t]);
    __threadfence();
    unsigned prev = 0;
    if (lane == 0) prev = atomicAdd(&P.gdone[g], 1u);
    prev = __shfl_sync(0xffffffffu, prev, 0);
    if (prev == nparts - 1) {  // last part to finish: combine in fixed order 0..s-1
      __threadfence();
      const float4 *base = P.part + (slot - part) * GS;
#pragma unroll
      for (int t = 0; t < TPL; ++t) {
        float hi[4] = {0.f, 0.f, 0.f, 0.f}, lo[4] = {0.f, 0.f, 0.f, 0.f};
        for (unsigned q = 0; q < nparts; ++q) {
          const float4 v = __ldcg(&base[(size_t)q * GS + lane + 32u * t]);
          two_sum_fold(hi[0], lo[0], v.x); two_sum_fold(hi[1], lo[1], v.y);
          two_sum_fold(hi[2], lo[2], v.z); two_sum_fold(hi[3], lo[3], v.w);
        }
        unsigned j = lane + 32u * t;
        if (j < gsize) {
          const float4 sum = make_float4(__fadd_rn(hi[0], lo[0]), __fadd_rn(hi[1], lo[1]), __fadd_rn(hi[2], lo[2]),
                                         __fadd_rn(hi[3], lo[3]));
          P.sacc[g0 + j] = sum;
          for (int q = 0; q < P.n_peers; ++q) P.peer_sacc[q][g0 + j] = sum;
          if (P.svel) kick_slot(P.svel + g0 + j, sum, P.kick_hdt);
          if (P.order) emit_caller(P, g0 + j, sum);
        }
      }
      if (P.n_peers > 0 && lane == 0) {  // every part's counts were added before it signalled gdone
        const uint2 c = __ldcg(&P.gcount[g]);
        for (int q = 0; q < P.n_peers; ++q) P.peer_gcount[q][g] = c;
      }
    }
  }
}

template <int TPL, bool COUNT, bool REL>
__global__ void __launch_bounds__(WALK_WARPS * 32, COUNT ? COUNT_MINB : walk_minb(TPL)) walk_force_kernel(const WalkParams P) {
  __shared__ WarpSmem smem[WALK_WARPS];
  WarpSmem &ws = smem[threadIdx.x >> 5];
  const int lane = threadIdx.x & 31;
  if (P.info->cells_overflow) return;  // a failed asynchronous rebuild: there is no tree to walk (tree.h)
  if (COUNT && (P.reuse_mode == 1 || (P.reuse_mode == 2 && P.info->reuse_costs))) return;  // costs come from the previous pass
  const unsigned n_items = COUNT ? P.n_groups : P.info->n_tasks;

  for (;;) {
    unsigned item = 0;
    if (lane == 0) item = atomicAdd(COUNT ? &P.info->group_ticket : &P.info->task_ticket, 1u);
    item = __shfl_sync(0xffffffffu, item, 0);
    if (item >= n_items) break;
    if (COUNT) {
      walk_task<TPL, true, REL>(P, ws, lane, item, item, 0u, 1u, 0ull);
      continue;
    }
    unsigned long long t_start;
    asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t_start));
    const unsigned tk = P.tasks[item];
    if (tk == TASK_NONE) continue;  // hole in the tail region of the task list
    const unsigned g = tk & TASK_GROUP_MASK, part = tk >> TASK_GROUP_BITS;
    const unsigned nparts = P.gparts[g] & PARTS_MASK;
    walk_task<TPL, false, REL>(P, ws, lane, item, g, part, nparts, t_start);
  }
}

// ------------------------------------------------------------------------------------------
// Task list (scheduling only; results depend on it only through the fixed-order partial sums).
// cost(g) = 13 n_pp + 37 n_pc, estimated by the truncated counting walk or taken from the previous pass's exact
// counts (tree_leapfrog). Task list of the groups this context walks (all of them unless the pass is sharded):
//   head : parts of EXPENSIVE groups (cost > 2 x mean over all groups: s = ceil(cost / mean) parts); in passes scheduled
//          by the previous pass's counts also, as single tasks, SUSPECT runs whose cost that pass cannot know, and, cut
//          into 16 parts, runs whose box is a large part of the system (task_cost_kernel); they start first
//   body : one task per ordinary group, in Peano-Hilbert order (L1/L2 locality between warps)
//   tail : the last n_tail groups, TAIL_PARTS parts each, so that the kernel ends on small tasks
// ------------------------------------------------------------------------------------------
constexpr double SPLIT_FINE = 1.0;  // parts per mean-cost unit of an expensive group
constexpr double SPLIT_AT = 2.0;      // a group is expensive above this multiple of the mean cost
constexpr unsigned MAX_PARTS = 63;
constexpr double BIG_BOX = 0.35;  // a run's box diagonal against the bounding box's (task_cost_kernel)
constexpr unsigned BIG_PARTS = 16;
constexpr double SUSPECT_AT = 3.0;  // a run's box diagonal against its neighbours' (task_cost_kernel)
constexpr unsigned TAIL_PARTS = 4;
constexpr long long TAIL_PER_SM = 16;  // groups per SM at the end of the list that are cut into TAIL_PARTS

__global__ void walk_reset_kernel(DevInfo *info, unsigned n_groups) {
  if (threadIdx.x == 0) {
    info->group_ticket = 0; info->task_ticket = 0; info->n_pp = 0; info->n_pc = 0; info->n_tasks = 0;
    info->sched_cost = 0;  // summed by the counting walk, or by group_cost_kernel from the previous pass's counts
    info->walk_overflow = 0;
    info->g_lo = 0; info->g_hi = n_groups;  // narrowed by shard_bounds_kernel in a sharded pass
    unsigned long long now;
    asm volatile("mov.u64 %0, %globaltimer;" : "=l"(now));
    info->t0_ns = now;
  }
}

__device__ __forceinline__ double prev_cost(const uint2 *__restrict__ gcount, unsigned g) {
  const uint2 c = gcount[g];
  return 13.0 * (double)c.x + 37.0 * (double)c.y;
}

// Cost estimate of every group for this pass (unit: 13 n_pp + 37 n_pc): the counting walk's (left in gdone), or --
// tree_leapfrog, the same particles one step later -- the exact counts of the previous pass (the neighbours cover a
// shift of the runs by up to two); in that case their sum is formed here.
__device__ __forceinline__ bool reuse_decided(int mode, const DevInfo *info) {
  return mode == 1 || (mode == 2 && info->reuse_costs);
}

__global__ void __launch_bounds__(256) group_cost_kernel(unsigned n_groups, DevInfo *info, const uint32_t *__restrict__ gdone,
                                                         const uint2 *__restrict__ prev_counts, int reuse_mode,
                                                         double *__restrict__ gcost) {
  const unsigned g = blockIdx.x * blockDim.x + threadIdx.x;
  const uint2 *prev = reuse_decided(reuse_mode, info) ? prev_counts : nullptr;  // block-uniform
  double own = 0.0;
  if (g < n_groups) {
    double cost;
    if (prev) {
      own = prev_cost(prev, g);
      cost = own;
      const unsigned a = g >= 2 ? g - 2 : 0u, b = g + 2 < n_groups ? g + 2 : n_groups - 1;
      for (unsigned q = a; q <= b; ++q) cost = fmax(cost, prev_cost(prev, q));
    } else {
      cost = (double)gdone[g];
    }
    gcost[g] = cost;
  }
  if (prev) {  // block-uniform
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) own += __shfl_xor_sync(0xffffffffu, own, o);
    __shared__ double s_own[8];
    if ((threadIdx.x & 31) == 0) s_own[threadIdx.x >> 5] = own;
    __syncthreads();
    if (threadIdx.x == 0) {
      double a = 0.0;
      for (int k = 0; k < 8; ++k) a += s_own[k];
      atomicAdd(&info->sched_cost, (unsigned long long)a);  // integers below 2^53: exact, order-independent
    }
  }
}

// Sharded pass: rank r of `world` walks the groups [B(r), B(r+1)), B(r) = number of groups whose exclusive
// cost prefix is below floor(total r / world) (contiguous pieces of the PH curve; L107:
// balanced on the flops of the tree-walk).  Costs are integers (13 n_pp + 37 n_pc), so the prefix sums do
// not depend on the order of addition and every context arrives at the same bounds.
constexpr int PART_BLOCK = 1024;  // groups per partial sum
__global__ void __launch_bounds__(256) shard_blocksum_kernel(unsigned n_groups, const double *__restrict__ gcost,
                                                             unsigned long long *__restrict__ bsum) {
  unsigned long long v = 0;
  const unsigned base = blockIdx.x * PART_BLOCK;
#pragma unroll
  for (int k = 0; k < PART_BLOCK / 256; ++k) {
    const unsigned g = base + k * 256 + threadIdx.x;
    if (g < n_groups) v += (unsigned long long)gcost[g];
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  __shared__ unsigned long long s[8];
  if ((threadIdx.x & 31) == 0) s[threadIdx.x >> 5] = v;
  __syncthreads();
  if (threadIdx.x == 0) {
    unsigned long long a = 0;
    for (int k = 0; k < 8; ++k) a += s[k];
    bsum[blockIdx.x] = a;
  }
}

// exclusive scan over the 1024 threads of a block (warp shuffles + one shared-memory step); also the total
__device__ __forceinline__ unsigned long long block_excl_scan_u64(unsigned long long v, unsigned long long *s_warp,
                                                                  unsigned long long &total) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  unsigned long long incl = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const unsigned long long n = __shfl_up_sync(0xffffffffu, incl, o);
    if (lane >= o) incl += n;
  }
  __syncthreads();  // s_warp may still be read from a previous call
  if (lane == 31) s_warp[w] = incl;
  __syncthreads();
  if (w == 0) {
    unsigned long long x = s_warp[lane], xi = x;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const unsigned long long n = __shfl_up_sync(0xffffffffu, xi, o);
      if (lane >= o) xi += n;
    }
    s_warp[lane] = xi - x;
    if (lane == 31) s_warp[32] = xi;
  }
  __syncthreads();
  total = s_warp[32];
  return s_warp[w] + incl - v;
}

__global__ void __launch_bounds__(PART_BLOCK) shard_bounds_kernel(unsigned n_groups, unsigned n_blocks,
                                                                  const double *__restrict__ gcost,
                                                                  const unsigned long long *__restrict__ bsum,
                                                                  unsigned rank, unsigned world, DevInfo *info) {
  __shared__ unsigned long long s_warp[33];
  __shared__ unsigned s_cnt;
  // 1. exclusive prefix of the partial sums at the start of this thread's chunk of them
  const unsigned chunk = (n_blocks + PART_BLOCK - 1) / PART_BLOCK;
  const unsigned b0 = min(threadIdx.x * chunk, n_blocks), b1 = min(b0 + chunk, n_blocks);
  unsigned long long mine = 0;
  for (unsigned b = b0; b < b1; ++b) mine += bsum[b];
  unsigned long long total;
  const unsigned long long start = block_excl_scan_u64(mine, s_warp, total);
  unsigned bound[2];
  for (int k = 0; k < 2; ++k) {
    const unsigned r = rank + k;
    const unsigned long long T = (total / world) * r + ((total % world) * r) / world;  // floor(total r / world)
    // 2. the last partial-sum block whose first group lies below T, and its exclusive prefix
    if (threadIdx.x == 0) s_cnt = 0u;
    __syncthreads();
    unsigned long long run = start;
    unsigned below = 0;
    for (unsigned b = b0; b < b1; ++b) { below += run < T; run += bsum[b]; }
    if (below) atomicAdd(&s_cnt, below);
    __syncthreads();
    const unsigned n_below = s_cnt;
    if (n_below == 0) { bound[k] = 0u; __syncthreads(); continue; }  // T = 0
    const unsigned bstar = n_below - 1;
    // exclusive prefix of block bstar = start of the thread that owns it + the blocks before it in that chunk
    __shared__ unsigned long long s_pre;
    if (bstar >= b0 && bstar < b1) {
      unsigned long long pre = start;
      for (unsigned b = b0; b < bstar; ++b) pre += bsum[b];
      s_pre = pre;
    }
    __syncthreads();
    // 3. inside that block: groups whose exclusive prefix is below T
    const unsigned g = bstar * PART_BLOCK + threadIdx.x;
    const unsigned long long c = g < n_groups ? (unsigned long long)gcost[g] : 0ull;
    unsigned long long dummy;
    const unsigned long long ex = s_pre + block_excl_scan_u64(c, s_warp, dummy);
    const int inside = __syncthreads_count(g < n_groups && ex < T);
    bound[k] = bstar * PART_BLOCK + (unsigned)inside;
  }
  if (threadIdx.x == 0) {
    info->g_lo = rank == 0 ? 0u : bound[0];
    info->g_hi = rank + 1 == world ? n_groups : bound[1];
  }
}

// The last groups of this context's range are cut into TAIL_PARTS parts so that the kernel ends on small
// tasks; a range shorter than that tail (small N, or many ranks sharing the pass) is cut entirely.  (Cutting
// finer does not pay: every part repeats the group's skeleton walk; 16 parts ran 2.5 x slower at N = 16,384.)
struct TailPlan { unsigned n_tail, parts; };
struct TailLimits { unsigned n_tail_max; };  // groups
__device__ __forceinline__ TailPlan tail_plan(const DevInfo *info, const TailLimits L) {
  TailPlan p;
  p.n_tail = min(L.n_tail_max, info->g_hi - info->g_lo);
  p.parts = TAIL_PARTS;
  return p;
}

__global__ void __launch_bounds__(256) task_cost_kernel(unsigned n_groups, const DevInfo *__restrict__ info,
                                                        uint32_t *__restrict__ a_cnt, uint32_t *__restrict__ gdone,
                                                        uint32_t *__restrict__ gthresh, const double *__restrict__ gcost,
                                                        const float *__restrict__ gbox, int reuse_mode, const TailLimits lim) {
  unsigned g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= n_groups) return;
  const float *suspect_gbox = reuse_decided(reuse_mode, info) ? gbox : nullptr;
  const unsigned tail_parts = tail_plan(info, lim).parts;
  const double mean = (double)info->sched_cost / (double)n_groups;  // over ALL groups, also in a sharded pass
  const double cost = gcost[g];
  const bool mine = g >= info->g_lo && g < info->g_hi;
  unsigned s = 0;
  if (mine && cost > SPLIT_AT * mean && mean > 0.0) {
    double want = ceil(SPLIT_FINE * cost / mean);
    s = want > (double)MAX_PARTS ? MAX_PARTS : (unsigned)want;
    if (s < 2) s = 0;
  }
  // The previous pass's counts (suspect_gbox != nullptr) cannot predict a group that has just become expensive: when
  // a far particle joins a run of 64, its box suddenly spans a dense region (measured at N = 33 M: 85 k -> 1.7 M cost
  // units from one step to the next, three such groups among 65 k, each a 5-7 ms task that ended one rank's kernel
  // 3-5 ms after the others on 8 ranks).  Such a run shows in its box: a diagonal more than SUSPECT_AT x the mean of
  // its four neighbours'.  It is listed at the front as one task, where its length cannot delay the end.
  if (mine && s == 0 && suspect_gbox && n_groups >= 5) {
    auto diag = [&](unsigned q) {
      const float *b = suspect_gbox + 6ull * q;
      const float dx = b[3] - b[0], dy = b[4] - b[1], dz = b[5] - b[2];
      return sqrtf(dx * dx + dy * dy + dz * dz);
    };
    const unsigned c = g < 2 ? 2u : (g + 2 >= n_groups ? n_groups - 3 : g);  // window centre kept inside the array
    float sum = 0.f;
    for (unsigned q = c - 2; q <= c + 2; ++q) if (q != g) sum += diag(q);
    if (diag(g) > (float)SUSPECT_AT * 0.25f * sum) s = 1;
  }
  // What the previous pass cannot predict at all is a run of far-apart particles (outskirts) whose box, already a large
  // part of the system, grows a little and now reaches into the dense centre: measured at N = 1 M, one step in ten had
  // such a run (box diagonal 54 -> 64, cost 0.75 -> 20 x the mean, neighbours unchanged), a single task of 9-20 ms in
  // a kernel of 8.2 ms.  Every run whose box diagonal exceeds BIG_BOX x the system's is therefore cut into BIG_PARTS parts
  // as if it cost BIG_PARTS x the mean (a few dozen runs; if they are cheap the parts are short).
  double assumed = cost;
  if (mine && s <= 1 && suspect_gbox) {
    const float *b = suspect_gbox + 6ull * g;
    const float dx = b[3] - b[0], dy = b[4] - b[1], dz = b[5] - b[2];
    const float sx = info->hi[0] - info->lo[0], sy = info->hi[1] - info->lo[1], sz = info->hi[2] - info->lo[2];
    if (dx * dx + dy * dy + dz * dz > (float)(BIG_BOX * BIG_BOX) * (sx * sx + sy * sy + sz * sz)) {
      s = BIG_PARTS;
      assumed = fmax(cost, (double)BIG_PARTS * mean);
    }
  }
  a_cnt[g] = s;
  gdone[g] = 0;
  // about 16 dealt entries per part: particles opened ~ cost / 13 (an over-estimate)
  const double per_entry = assumed / 13.0 / (16.0 * (s ? s : tail_parts));
  gthresh[g] = per_entry < 32.0 ? 32u : (per_entry > 1e9 ? 1000000000u : (unsigned)per_entry);
}

// after the exclusive scan of a_cnt (in place -> a_off): expensive groups that do not fit the
// partial-sum buffer (a suffix of them, offsets are monotone) fall back to one part; classifies
// every group of this context's range (head / body / tail) and writes the body counts
__global__ void __launch_bounds__(256) task_class_kernel(unsigned n_groups, const TailLimits lim,
                                                         const uint32_t *__restrict__ a_off, const uint32_t *a_total,
                                                         unsigned head_cap, uint8_t *__restrict__ gparts,
                                                         uint32_t *__restrict__ b_cnt, uint2 *__restrict__ gcount,
                                                         DevInfo *info) {
  unsigned g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= n_groups) return;
  const unsigned tot = *a_total;
  if (g == 0 && tot <= head_cap) info->n_tasks_a = tot;
  const unsigned lo = info->g_lo, hi = info->g_hi;
  if (g < lo || g >= hi) { gparts[g] = 1; b_cnt[g] = 0u; return; }  // another context's group: its counts arrive by peer store
  const TailPlan tp = tail_plan(info, lim);
  const unsigned n_tail = tp.n_tail;
  const unsigned off = a_off[g];
  const unsigned nxt = (g + 1 < n_groups) ? a_off[g + 1] : tot;
  unsigned s = nxt - off;
  if (s && nxt > head_cap) {
    if (off <= head_cap) info->n_tasks_a = off;  // the first expensive group that does not fit
    s = 0;
  }
  const bool tail = g >= hi - n_tail;
  gparts[g] = (uint8_t)(s ? (s | PARTS_HEAD) : (tail ? tp.parts : 1u));
  b_cnt[g] = (s || tail) ? 0u : 1u;
  gcount[g] = make_uint2(0u, 0u);
}

__global__ void __launch_bounds__(256) task_fill_kernel(unsigned n_groups, const TailLimits lim,
                                                        const uint32_t *__restrict__ a_off,
                                                        const uint32_t *__restrict__ b_off, const uint32_t *b_total,
                                                        const uint8_t *__restrict__ gparts, uint32_t *__restrict__ tasks,
                                                        DevInfo *info) {
  unsigned g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= n_groups) return;
  const unsigned lo = info->g_lo, hi = info->g_hi;
  const TailPlan tp = tail_plan(info, lim);
  const unsigned n_tail = tp.n_tail;
  const unsigned a_end = info->n_tasks_a;
  const unsigned tail_start = a_end + *b_total;
  if (g == 0) { info->n_tasks = tail_start + n_tail * tp.parts; info->tail_start = tail_start; }
  if (g < lo || g >= hi) return;
  const unsigned gp = gparts[g], s = gp & PARTS_MASK;
  const bool head = gp & PARTS_HEAD;
  const bool tail = g >= hi - n_tail;
  if (head) {
    const unsigned off = a_off[g];
    for (unsigned j = 0; j < s; ++j) tasks[off + j] = g | (j << TASK_GROUP_BITS);
  } else if (!tail) {
    tasks[a_end + b_off[g]] = g;
  }
  if (tail) {  // fixed slots; an expensive group inside the tail range leaves a hole here
    const unsigned base = tail_start + (g - (hi - n_tail)) * tp.parts;
    for (unsigned j = 0; j < tp.parts; ++j) tasks[base + j] = head ? TASK_NONE : (g | (j << TASK_GROUP_BITS));
  }
}

// a11: results to the caller's arrays (caller order), only when the caller gave any; the library itself keeps its
// state and results in slot order.  A gather through the inverse of `order` (slot_of, built once per sort): the random
// side is a 16-byte read, the writes are sequential (the scatter form, 12- and 4-byte random writes, ran at a third of
// the speed at N = 134 M).
__global__ void __launch_bounds__(256) gather_out_kernel(const float4 *__restrict__ sacc, const uint32_t *__restrict__ slot_of,
                                                         long long N, float *__restrict__ acc, float *__restrict__ pot) {
  long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (i >= N) return;
  const float4 a = sacc[slot_of[i]];
  if (acc) { acc[3 * i] = a.x; acc[3 * i + 1] = a.y; acc[3 * i + 2] = a.z; }
  if (pot) pot[i] = a.w;
}

// a12: the closing half kick of a step as its own pass (sharded passes: after the barrier; otherwise it is fused into the
// walk's epilogue, kick_slot): v = fma(a, dt/2, v), slot order, sequential
__global__ void __launch_bounds__(256) kick_kernel(float4 *__restrict__ svel, const float4 *__restrict__ sacc, long long N,
                                                   float hdt, const DevInfo *__restrict__ info) {
  long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (i >= N || info->cells_overflow) return;
  float4 v = svel[i];
  const float4 a = sacc[i];
  v.x = __fmaf_rn(a.x, hdt, v.x); v.y = __fmaf_rn(a.y, hdt, v.y); v.z = __fmaf_rn(a.z, hdt, v.z);
  svel[i] = v;
}

__global__ void energy_reset_kernel(DevInfo *info) {
  if (threadIdx.x == 0) { info->ekin = 0.0; info->epot = 0.0; }
}

__global__ void __launch_bounds__(256) energy_kernel(const float4 *__restrict__ spos, const float4 *__restrict__ svel,
                                                     const float4 *__restrict__ sacc, long long N, bool have_vel,
                                                     DevInfo *info) {
  double ke = 0.0, pe = 0.0;
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x) {
    const double m = (double)spos[i].w;
    if (have_vel) {
      const float4 v = svel[i];
      ke += 0.5 * m * ((double)v.x * v.x + (double)v.y * v.y + (double)v.z * v.z);
    }
    pe += 0.5 * m * (double)sacc[i].w;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    ke += __shfl_xor_sync(0xffffffffu, ke, o);
    pe += __shfl_xor_sync(0xffffffffu, pe, o);
  }
  __shared__ double s_k[8], s_p[8];
  if ((threadIdx.x & 31) == 0) { s_k[threadIdx.x >> 5] = ke; s_p[threadIdx.x >> 5] = pe; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double a = 0, b = 0;
    for (int k = 0; k < 8; ++k) { a += s_k[k]; b += s_p[k]; }
    atomicAdd(&info->ekin, a);
    atomicAdd(&info->epot, b);
  }
}

// the caller's velocities (caller order) into the slot-order state
__global__ void __launch_bounds__(256) set_vel_kernel(const float *__restrict__ v3, const uint32_t *__restrict__ order,
                                                      float4 *__restrict__ svel, long long N) {
  long long s = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (s >= N) return;
  const long long i = order[s];
  svel[s] = make_float4(v3[3 * i], v3[3 * i + 1], v3[3 * i + 2], 0.0f);
}

// the slot-order state and results to the caller's arrays (caller order)
__global__ void __launch_bounds__(256) get_state_kernel(const float4 *__restrict__ spos, const float4 *__restrict__ svel,
                                                        const float4 *__restrict__ sacc, const uint32_t *__restrict__ order,
                                                        long long N, float *__restrict__ pos, float *__restrict__ v3,
                                                        float *__restrict__ acc, float *__restrict__ pot) {
  long long s = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (s >= N) return;
  const long long i = order[s];
  if (pos) { float4 p = spos[s]; pos[3 * i] = p.x; pos[3 * i + 1] = p.y; pos[3 * i + 2] = p.z; }
  if (v3) { float4 v = svel[s]; v3[3 * i] = v.x; v3[3 * i + 1] = v.y; v3[3 * i + 2] = v.z; }
  if (acc || pot) {
    float4 a = sacc[s];
    if (acc) { acc[3 * i] = a.x; acc[3 * i + 1] = a.y; acc[3 * i + 2] = a.z; }
    if (pot) pot[i] = a.w;
  }
}

// slot of every caller index (tree_direct looks its targets up by caller index)
__global__ void __launch_bounds__(256) inverse_order_kernel(const uint32_t *__restrict__ order, long long N,
                                                            uint32_t *__restrict__ slot_of) {
  long long s = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (s < N) slot_of[order[s]] = (uint32_t)s;
}

// ------------------------------------------------------------------------------------------
// Direct summation (the definition the tree force approximates), FP64.
// One thread per target, sources staged through shared memory; the source range is cut over
// blockIdx.y and the partial sums are added with FP64 atomics (acc / pot zeroed before).
// ------------------------------------------------------------------------------------------
constexpr int DIRECT_THREADS = 128;

__global__ void __launch_bounds__(DIRECT_THREADS) direct_kernel(const float4 *__restrict__ posm, long long N,
                                                                const long long *__restrict__ idx,
                                                                const uint32_t *__restrict__ slot_of, long long n,
                                                                double eps2, double *__restrict__ acc,
                                                                double *__restrict__ pot) {
  __shared__ float4 tile[DIRECT_THREADS];
  const long long k = blockIdx.x * (long long)DIRECT_THREADS + threadIdx.x;
  const long long i = k < n ? (long long)slot_of[idx[k]] : -1;  // the sources are summed in slot order
  const float4 pi = i >= 0 ? posm[i] : make_float4(0.f, 0.f, 0.f, 0.f);
  const double xi = pi.x, yi = pi.y, zi = pi.z;
  const long long chunk = (N + gridDim.y - 1) / gridDim.y;
  const long long j0 = blockIdx.y * chunk, j1 = j0 + chunk < N ? j0 + chunk : N;
  double ax = 0.0, ay = 0.0, az = 0.0, ph = 0.0;
  for (long long base = j0; base < j1; base += DIRECT_THREADS) {
    const long long j = base + threadIdx.x;
    tile[threadIdx.x] = j < j1 ? posm[j] : make_float4(0.f, 0.f, 0.f, 0.f);
    __syncthreads();
    const int cnt = (int)(j1 - base < DIRECT_THREADS ? j1 - base : DIRECT_THREADS);
#pragma unroll 4
    for (int q = 0; q < cnt; ++q) {
      const float4 s = tile[q];
      const double dx = (double)s.x - xi, dy = (double)s.y - yi, dz = (double)s.z - zi;
      const double r2 = dx * dx + dy * dy + dz * dz + eps2;
      const double m = (base + q == i) ? 0.0 : (double)s.w;  // self term skipped by index (S2)
      const double ri = (base + q == i) ? 0.0 : rsqrt(r2);
      const double mr = m * ri, mr3 = mr * ri * ri;
      ax += mr3 * dx; ay += mr3 * dy; az += mr3 * dz; ph -= mr;
    }
    __syncthreads();
  }
  if (i >= 0) {
    atomicAdd(&acc[3 * k], ax); atomicAdd(&acc[3 * k + 1], ay); atomicAdd(&acc[3 * k + 2], az);
    atomicAdd(&pot[k], ph);
  }
}

// ------------------------------------------------------------------------------------------
// Measurement aid: the FP32 FMA rate this GPU sustains on register operands, the measured
// denominator beside the nominal peak of the roofline.  Eight independent FFMA chains per thread with one
// fresh register operand each (multiplier and addend repeat, so they come from the operand-reuse cache /
// immediates): the form that reaches one FFMA per clock and scheduler.
// ------------------------------------------------------------------------------------------
constexpr int PEAK_THREADS = 256, PEAK_CHAINS = 8, PEAK_UNROLL = 32;
__global__ void __launch_bounds__(PEAK_THREADS) fp32_peak_kernel(float *out, int iters, float mul, float add) {
  float a[PEAK_CHAINS];
#pragma unroll
  for (int k = 0; k < PEAK_CHAINS; ++k) a[k] = (float)(threadIdx.x + k) * 1e-3f;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < PEAK_UNROLL; ++u) {
#pragma unroll
      for (int k = 0; k < PEAK_CHAINS; ++k) a[k] = fmaf(a[k], mul, add);
    }
  }
  float s = 0.f;
#pragma unroll
  for (int k = 0; k < PEAK_CHAINS; ++k) s += a[k];
  if (s == 123.456f) out[0] = s;  // never true for these inputs; keeps the chains alive
}

int run_fp32_peak(tree_ctx *t, double *tflops) {
  cudaEvent_t e0, e1;
  BH_CUDA(cudaEventCreate(&e0));
  BH_CUDA(cudaEventCreate(&e1));
  const int blocks = t->sm_count * 8, iters = 512;
  float *sink = reinterpret_cast<float *>(t->d_hlut);  // never written (see the kernel)
  double best = 0.0;
  for (int rep = 0; rep < 4; ++rep) {  // first repetition warms up
    cudaEventRecord(e0, t->stream);
    fp32_peak_kernel<<<blocks, PEAK_THREADS, 0, t->stream>>>(sink, iters, 0.999999f, 1e-7f);
    cudaEventRecord(e1, t->stream);
    cudaError_t e = cudaEventSynchronize(e1);
    if (e != cudaSuccess) { cudaEventDestroy(e0); cudaEventDestroy(e1); return set_err(t, TREE_ERR_CUDA, "fp32_peak", e); }
    t->launches++;
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    const double flop = 2.0 * PEAK_CHAINS * PEAK_UNROLL * (double)iters * PEAK_THREADS * (double)blocks;
    if (rep > 0 && ms > 0.f) best = fmax(best, flop / (ms * 1e-3) / 1e12);
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  *tflops = best;
  return 0;
}

// ------------------------------------------------------------------------------------------
// host launchers
// ------------------------------------------------------------------------------------------
static inline unsigned blocks_for(long long n, int threads) { return (unsigned)((n + threads - 1) / threads); }

int run_opening(tree_ctx *t, float theta) {
  opening_kernel<<<blocks_for(t->cells_bound, 256), 256, 0, t->stream>>>(
      t->d_info, theta, t->b.c_level, t->b.c_cm, t->b.c_qa, t->mac == TREE_MAC_BMAX ? t->b.c_tlo : nullptr, t->b.c_test,
      t->rel_on && t->amag_valid ? t->b.c_q : nullptr);
  BH_LAUNCH_CHECK("opening");
  return 0;
}

// Relative criterion (tree_set_mac_relative): |a| per slot, one IEEE operation each in this order, and the group's scale
// alpha * min |a| (one warp per group; min is exact, one multiplication).
__global__ void __launch_bounds__(256) amag_acc_kernel(const float4 *__restrict__ sacc, long long N, float *__restrict__ amag) {
  long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (i >= N) return;
  const float4 a = sacc[i];
  amag[i] = __fsqrt_rn(__fmaf_rn(a.z, a.z, __fmaf_rn(a.y, a.y, __fmul_rn(a.x, a.x))));
}

__global__ void __launch_bounds__(256) amag_caller_kernel(const float *__restrict__ given, const uint32_t *__restrict__ order,
                                                          long long N, float *__restrict__ amag) {
  long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (i < N) amag[i] = given[order[i]];
}

__global__ void __launch_bounds__(256) group_scale_kernel(const float *__restrict__ amag, long long N, int group, float alpha,
                                                          long long n_groups, float *__restrict__ gscale) {
  const long long g = (blockIdx.x * (long long)blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (g >= n_groups) return;
  const long long s0 = g * group;
  float m = INFINITY;
  for (int j = lane; j < group; j += 32)
    if (s0 + j < N) m = fminf(m, amag[s0 + j]);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = fminf(m, __shfl_xor_sync(0xffffffffu, m, o));
  if (lane == 0) gscale[g] = __fmul_rn(alpha, m);
}

int run_amag_from_acc(tree_ctx *t) {
  amag_acc_kernel<<<blocks_for(t->N, 256), 256, 0, t->stream>>>(t->b.sacc, t->N, t->b.amag2[t->cur]);
  BH_LAUNCH_CHECK("amag_acc");
  return 0;
}

int run_amag_from_caller(tree_ctx *t, const float *amag) {
  amag_caller_kernel<<<blocks_for(t->N, 256), 256, 0, t->stream>>>(amag, t->b.order, t->N, t->b.amag2[t->cur]);
  BH_LAUNCH_CHECK("amag_caller");
  return 0;
}

int run_group_scale(tree_ctx *t) {
  group_scale_kernel<<<blocks_for(t->n_groups * 32, 256), 256, 0, t->stream>>>(t->b.amag2[t->cur], t->N, t->group, t->rel_alpha,
                                                                               t->n_groups, t->b.gscale);
  BH_LAUNCH_CHECK("group_scale");
  return 0;
}

// Is this build the particle set of the previous force pass, moved a little?  Counts, among up to 65,536 sampled groups,
// those whose box centre lies outside the hull of the previous pass's boxes of the runs g-W..g+W, or whose box is not
// finite.  (Particles that change their place in the Peano-Hilbert order shift every run between their old and new place
// by one particle, so run g of this build is some run near g of the last one; the net shift grows like sqrt(N):
// W = max(8, sqrt(N) / 128).)  Scheduling hint only.
__global__ void __launch_bounds__(256) box_moved_kernel(unsigned n_groups, unsigned n_samples, unsigned stride, unsigned window,
                                                        const float *__restrict__ gbox, const float *__restrict__ gbox_prev,
                                                        DevInfo *info) {
  const unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
  bool moved = false;
  if (i < n_samples) {
    const unsigned g = i * stride;
    const float *a = gbox + 6ull * g;
    const float cx = 0.5f * (a[0] + a[3]), cy = 0.5f * (a[1] + a[4]), cz = 0.5f * (a[2] + a[5]);
    const unsigned q0 = g >= window ? g - window : 0u;
    const unsigned q1 = g + window < n_groups ? g + window : n_groups - 1u;
    float lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY};
    for (unsigned q = q0; q <= q1; ++q) {
      const float *b = gbox_prev + 6ull * q;
#pragma unroll
      for (int c = 0; c < 3; ++c) { lo[c] = fminf(lo[c], b[c]); hi[c] = fmaxf(hi[c], b[3 + c]); }
    }
    moved = !(cx >= lo[0] && cx <= hi[0] && cy >= lo[1] && cy <= hi[1] && cz >= lo[2] && cz <= hi[2]);
  }
  const unsigned m = __ballot_sync(0xffffffffu, moved);
  if ((threadIdx.x & 31) == 0 && m) atomicAdd(&info->moved_groups, (unsigned)__popc(m));
}

__global__ void box_decide_kernel(unsigned n_samples, DevInfo *info) {
  // measured: 0-2 % of the sampled runs moved for a drifted set, 99.7 % for an unrelated one
  if (threadIdx.x == 0) info->reuse_costs = (unsigned long long)info->moved_groups * 8ull <= n_samples ? 1u : 0u;
}

// Decides on the device (info->reuse_costs) whether this pass schedules by the previous pass's counts: no read-back.
int run_box_check(tree_ctx *t) {
  const unsigned ng = (unsigned)t->n_groups;
  const unsigned stride = (ng + 65535u) / 65536u, ns = (ng + stride - 1u) / stride;
  const unsigned window = std::max(8u, (unsigned)(std::sqrt((double)t->N) / 128.0));
  BH_CUDA(cudaMemsetAsync(&t->d_info->moved_groups, 0, sizeof(unsigned), t->stream));
  box_moved_kernel<<<(ns + 255) / 256, 256, 0, t->stream>>>(ng, ns, stride, window, t->b.gbox, t->b.gbox_prev, t->d_info);
  BH_LAUNCH_CHECK("box_moved");
  box_decide_kernel<<<1, 32, 0, t->stream>>>(ns, t->d_info);
  BH_LAUNCH_CHECK("box_decide");
  return 0;
}

template <int TPL, bool REL>
static int launch_walk(tree_ctx *t, const WalkParams &P, unsigned grid) {
  const unsigned ng = P.n_groups, gb = (ng + 255) / 256;
  DevInfo *info = t->d_info;
  uint32_t *tot = info->sched_tot;
  // 1. cost of every group: the walk without the evaluation, or the previous pass's exact counts
  const int mode = P.reuse_mode;
  if (mode != 1) {  // mode 2: the kernel returns at once if the device decided to reuse the previous counts
    const long long cwant = (ng + WALK_WARPS - 1) / WALK_WARPS, ccap = (long long)t->sm_count * COUNT_MINB;
    walk_force_kernel<TPL, true, REL><<<(unsigned)(cwant < ccap ? cwant : ccap), WALK_WARPS * 32, 0, t->stream>>>(P);
    BH_LAUNCH_CHECK("walk_count");
  }
  group_cost_kernel<<<gb, 256, 0, t->stream>>>(ng, info, t->b.gdone, t->b.gcount2[(t->pass + 1) & 1], mode, t->b.gcost);
  BH_LAUNCH_CHECK("group_cost");
  if (t->shard_world > 1) {
    const unsigned nb = (ng + PART_BLOCK - 1) / PART_BLOCK;  // <= 2^16: sched_b (one word per group) has room
    unsigned long long *bsum = reinterpret_cast<unsigned long long *>(t->b.sched_b);
    shard_blocksum_kernel<<<nb, 256, 0, t->stream>>>(ng, t->b.gcost, bsum);
    BH_LAUNCH_CHECK("shard_blocksum");
    shard_bounds_kernel<<<1, PART_BLOCK, 0, t->stream>>>(ng, nb, t->b.gcost, bsum, (unsigned)t->shard_rank,
                                                         (unsigned)t->shard_world, info);
    BH_LAUNCH_CHECK("shard_bounds");
  }
  // 2. task list of this context's range: split expensive groups, longest work first
  TailLimits lim;
  lim.n_tail_max = (unsigned)std::min<long long>(TAIL_PER_SM * t->sm_count, t->tail_cap / (long long)TAIL_PARTS);
  task_cost_kernel<<<gb, 256, 0, t->stream>>>(ng, info, t->b.sched_a, t->b.gdone, t->b.gthresh, t->b.gcost,
                                              t->b.gbox, mode, lim);
  BH_LAUNCH_CHECK("task_cost");
  int rc = device_excl_scan(t, t->b.sched_a, ng, tot);
  if (rc) return rc;
  task_class_kernel<<<gb, 256, 0, t->stream>>>(ng, lim, t->b.sched_a, tot, (unsigned)t->head_cap, t->b.gparts,
                                               t->b.sched_b, t->b.gcount, info);
  BH_LAUNCH_CHECK("task_class");
  rc = device_excl_scan(t, t->b.sched_b, ng, tot + 1);
  if (rc) return rc;
  task_fill_kernel<<<gb, 256, 0, t->stream>>>(ng, lim, t->b.sched_a, t->b.sched_b, tot + 1, t->b.gparts, t->b.tasks,
                                              info);
  BH_LAUNCH_CHECK("task_fill");
  if (t->ev_valid[EV_SCHED]) cudaEventRecord(t->ev[EV_SCHED], t->stream);
  // 3. the fused walk + force over the task list
  walk_force_kernel<TPL, false, REL><<<grid, WALK_WARPS * 32, 0, t->stream>>>(P);
  BH_LAUNCH_CHECK("walk_force");
  return 0;
}

int run_walk(tree_ctx *t, float eps, float kick_hdt, float *out_acc, float *out_pot) {
  WalkParams P;
  P.reuse_mode = t->reuse_mode;
  const bool fuse_out = (out_acc || out_pot) && t->shard_world <= 1;  // sharded: most results arrive from peers (force_end gathers)
  P.order = fuse_out ? t->b.order : nullptr;
  P.out_acc = out_acc; P.out_pot = out_pot;
  const bool fuse_kick = kick_hdt != 0.0f && t->shard_world <= 1;
  P.svel = fuse_kick ? t->b.svel : nullptr;
  P.kick_hdt = kick_hdt;
  P.spos = t->b.spos; P.c_test = t->b.c_test; P.c_link = t->b.c_link;
  P.c_cm = t->b.c_cm; P.c_qa = t->b.c_qa; P.c_qb = t->b.c_qb;
  P.gbox = t->b.gbox; P.sacc = t->b.sacc; P.gcount = t->b.gcount; P.info = t->d_info;
  P.n_peers = 0;
  for (int r = 0; r < TREE_SHARD_MAX_WORLD; ++r) { P.peer_sacc[r] = nullptr; P.peer_gcount[r] = nullptr; }
  if (t->shard_world > 1)
    for (int r = 0; r < t->shard_world; ++r)
      if (r != t->shard_rank) {
        shard_views(t, t->peer_base[r], (int)(t->pass & 1), &P.peer_sacc[P.n_peers], &P.peer_gcount[P.n_peers]);
        ++P.n_peers;
      }
  P.c_count = t->b.c_count; P.trace = t->b.trace; P.gthresh = t->b.gthresh; P.tasks = t->b.tasks; P.gparts = t->b.gparts; P.gdone = t->b.gdone; P.part = t->b.part;
  P.N = t->N; P.n_groups = (unsigned)t->n_groups; P.eps2 = eps * eps;
  walk_reset_kernel<<<1, 32, 0, t->stream>>>(t->d_info, (unsigned)t->n_groups);
  BH_LAUNCH_CHECK("walk_reset");
  long long want = (t->n_groups + WALK_WARPS - 1) / WALK_WARPS;
  long long cap = (long long)t->sm_count * walk_minb(t->group / 32);
  unsigned grid = (unsigned)(want < cap ? want : cap);
  if (t->ev_valid[EV_OPEN]) cudaEventRecord(t->ev[EV_OPEN], t->stream);
  int rc;
  const bool rel = t->rel_on && t->amag_valid;  // no |a| yet (first pass after tree_build): the geometric criterion alone
  P.c_q = rel ? t->b.c_q : nullptr; P.gscale = rel ? t->b.gscale : nullptr;
  switch (t->group) {
    case 32: rc = rel ? launch_walk<1, true>(t, P, grid) : launch_walk<1, false>(t, P, grid); break;
    case 64: rc = rel ? launch_walk<2, true>(t, P, grid) : launch_walk<2, false>(t, P, grid); break;
    case 128: rc = rel ? launch_walk<4, true>(t, P, grid) : launch_walk<4, false>(t, P, grid); break;
    default: return set_err(t, TREE_ERR_ARG, "group size");
  }
  if (rc) return rc;
  if (t->ev_valid[EV_WALK]) cudaEventRecord(t->ev[EV_WALK], t->stream);
  return 0;
}

// slot of every caller index, in the key buffer that does not hold the sorted keys (free between two sorts)
static int ensure_slot_of(tree_ctx *t, uint32_t **slot_of) {
  *slot_of = reinterpret_cast<uint32_t *>(t->b.key[t->sorted ^ 1]);
  if (t->slot_of_valid) return 0;
  inverse_order_kernel<<<blocks_for(t->N, 256), 256, 0, t->stream>>>(t->b.order, t->N, *slot_of);
  BH_LAUNCH_CHECK("inverse_order");
  t->slot_of_valid = true;
  return 0;
}

int run_scatter_out(tree_ctx *t, float *acc, float *pot) {
  if (!acc && !pot) return 0;
  uint32_t *slot_of;
  int rc = ensure_slot_of(t, &slot_of);
  if (rc) return rc;
  gather_out_kernel<<<blocks_for(t->N, 256), 256, 0, t->stream>>>(t->b.sacc, slot_of, t->N, acc, pot);
  BH_LAUNCH_CHECK("gather_out");
  return 0;
}

int run_kick(tree_ctx *t, float dt) {
  kick_kernel<<<blocks_for(t->N, 256), 256, 0, t->stream>>>(t->b.svel, t->b.sacc, t->N, 0.5f * dt, t->d_info);
  BH_LAUNCH_CHECK("kick");
  return 0;
}

int run_energy(tree_ctx *t) {
  energy_reset_kernel<<<1, 32, 0, t->stream>>>(t->d_info);
  BH_LAUNCH_CHECK("energy_reset");
  long long want = (t->N + 255) / 256, cap = (long long)t->sm_count * 8;
  energy_kernel<<<(unsigned)(want < cap ? want : cap), 256, 0, t->stream>>>(t->b.spos, t->b.svel, t->b.sacc, t->N,
                                                                          t->have_vel, t->d_info);
  BH_LAUNCH_CHECK("energy");
  return 0;
}

int run_set_velocity(tree_ctx *t, const float *vel) {
  set_vel_kernel<<<blocks_for(t->N, 256), 256, 0, t->stream>>>(vel, t->b.order, t->b.svel, t->N);
  BH_LAUNCH_CHECK("set_velocity");
  return 0;
}

int run_direct(tree_ctx *t, const long long *idx, long long n, float eps, double *acc, double *pot) {
  cudaError_t e = cudaMemsetAsync(acc, 0, (size_t)n * 3 * sizeof(double), t->stream);
  if (e == cudaSuccess) e = cudaMemsetAsync(pot, 0, (size_t)n * sizeof(double), t->stream);
  if (e != cudaSuccess) return set_err(t, TREE_ERR_CUDA, "tree_direct: memset", e);
  uint32_t *slot_of;
  int rc = ensure_slot_of(t, &slot_of);
  if (rc) return rc;
  const unsigned gx = blocks_for(n, DIRECT_THREADS);
  long long gy = ((long long)t->sm_count * 16 + gx - 1) / gx;  // about 16 blocks per SM in total
  const long long gy_max = (t->N + 4 * DIRECT_THREADS - 1) / (4 * DIRECT_THREADS);
  if (gy > gy_max) gy = gy_max;
  if (gy < 1) gy = 1;
  if (gy > 65535) gy = 65535;
  direct_kernel<<<dim3(gx, (unsigned)gy), DIRECT_THREADS, 0, t->stream>>>(t->b.spos, t->N, idx, slot_of, n,
                                                                          (double)eps * (double)eps, acc, pot);
  BH_LAUNCH_CHECK("direct");
  return 0;
}

int run_get_state(tree_ctx *t, float *pos, float *vel, float *acc, float *pot) {
  get_state_kernel<<<blocks_for(t->N, 256), 256, 0, t->stream>>>(t->b.spos, t->b.svel, t->b.sacc, t->b.order, t->N, pos, vel,
                                                                 acc, pot);
  BH_LAUNCH_CHECK("get_state");
  return 0;
}

}  // namespace bh
