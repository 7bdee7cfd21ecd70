// Measurement aid (sm_100a), not on the product path: the walk and the evaluation of a force pass as TWO kernels, with the
// interaction lists going through global memory.  tree_measure_listeval times both on the tree and theta of the last force
// pass: the evaluation alone is the upper bound of what separating walker and evaluator warps in the fused kernel
// could reach; the walk alone is what would have to be hidden.  A translation unit of its own, so
// that the code placement of the fused kernel's module does not depend on it.
#include <vector>

#include "bh_eval.cuh"

// Kernel W walks every group (one warp each, the walk of the fused kernel without evaluation) and writes its interaction
// lists to global memory: accepted cell ids, particle indices of opened leaves.  Kernel E evaluates the lists with the
// fused kernel's evaluators and nothing else.  Groups are handed out in descending cost (one warp per group, no splitting:
// meaningful where no single group is a sizeable part of the pass, N >= 8 M).
namespace bh {

struct ListParams {
  WalkParams P;
  const uint32_t *gorder;   // groups in the order they are handed out
  const uint32_t *pc_off, *pp_off;  // first entry of each group's (32-padded) lists
  uint32_t *pc_list, *pp_list;
  float4 *out;              // E: results (slot order)
  unsigned *ticket;
};

__global__ void __launch_bounds__(WALK_WARPS * 32, COUNT_MINB) walk_lists_kernel(const ListParams L) {
  __shared__ WarpSmem smem[WALK_WARPS];
  WarpSmem &ws = smem[threadIdx.x >> 5];
  const WalkParams &P = L.P;
  const int lane = threadIdx.x & 31;
  const unsigned lt = (1u << lane) - 1u;
  const unsigned gt = ~((lt << 1) | 1u);
  for (;;) {
    unsigned item = 0;
    if (lane == 0) item = atomicAdd(L.ticket, 1u);
    item = __shfl_sync(0xffffffffu, item, 0);
    if (item >= P.n_groups) break;
    const unsigned g = L.gorder[item];
    const float *gb = P.gbox + 6ll * g;
    const float bx0 = gb[0], by0 = gb[1], bz0 = gb[2], bx1 = gb[3], by1 = gb[4], bz1 = gb[5];
    uint32_t *pc_out = L.pc_list + L.pc_off[g], *pp_out = L.pp_list + L.pp_off[g];
    int sp = 1, pc_pending = 0, pp_entries = 0, pp_pending = 0;
    unsigned pc_written = 0, pp_written = 0;
    if (lane == 0) ws.stack[0] = 0u;
    __syncwarp();
    auto flush_pp = [&](int want) {  // `want` particle indices from the back of the range queue to the list
      const bool have = lane < pp_entries;
      uint2 e = have ? ws.ppq[pp_entries - 1 - lane] : make_uint2(0u, 0u);
      const unsigned n = have ? min(e.y, 33u) : 0u;
      const unsigned incl = warp_incl_scan_u(n, lane), excl = incl - n;
      const bool take = have && excl < (unsigned)want;
      const bool full = incl <= (unsigned)want;
      if (take && !full) { unsigned k = (unsigned)want - excl; ws.ppq[pp_entries - 1 - lane] = make_uint2(e.x + k, e.y - k); }
      pp_entries -= __popc(__ballot_sync(0xffffffffu, take && full));
      const unsigned head = __reduce_or_sync(0xffffffffu, take ? (1u << excl) : 0u);
      const int ei = __popc(head & (0xffffffffu >> (31 - lane))) - 1;
      const unsigned fx = __shfl_sync(0xffffffffu, e.x, ei & 31);
      const unsigned ex = __shfl_sync(0xffffffffu, excl, ei & 31);
      if (lane < want) pp_out[pp_written + lane] = fx + ((unsigned)lane - ex);
      pp_written += want;
      __syncwarp();
    };
    while (sp > 0) {
      const bool have = lane < sp;
      const int my = sp - 1 - lane;
      const unsigned e = have ? ws.stack[my] : 0u;
      const unsigned n = have ? (e & 7u) + 1u : 0u;
      const unsigned incl = warp_incl_scan_u(n, lane), excl = incl - n;
      const bool take = have && excl < 32u;
      const bool full = incl <= 32u;
      if (take && !full) { unsigned k = 32u - excl; ws.stack[my] = (((e >> 3) + k) << 3) | (n - k - 1u); }
      sp -= __popc(__ballot_sync(0xffffffffu, take && full));
      const unsigned tot_all = __shfl_sync(0xffffffffu, incl, 31);
      const unsigned total = tot_all < 32u ? tot_all : 32u;
      const unsigned head = __reduce_or_sync(0xffffffffu, take ? (1u << excl) : 0u);
      const int ei = __popc(head & (0xffffffffu >> (31 - lane))) - 1;
      const unsigned fx = __shfl_sync(0xffffffffu, e >> 3, ei & 31);
      const unsigned ex = __shfl_sync(0xffffffffu, excl, ei & 31);
      const bool valid = (unsigned)lane < total;
      const unsigned cell = fx + ((unsigned)lane - ex);
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
        const bool leaf = !(lk.y & LEAF_FLAG);
        open_leaf = !accept && leaf;
        open_int = !accept && !leaf;
      }
      {
        const unsigned m = __ballot_sync(0xffffffffu, open_int);
        if (open_int) ws.stack[sp + __popc(m & gt)] = (lk.x << 3) | ((lk.y & 0xfu) - 1u);
        sp += __popc(m);
      }
      {
        const unsigned m = __ballot_sync(0xffffffffu, accept);
        if (accept) ws.pcq[pc_pending + __popc(m & lt)] = cell;
        pc_pending += __popc(m);
      }
      {
        const unsigned m = __ballot_sync(0xffffffffu, open_leaf);
        if (open_leaf) ws.ppq[pp_entries + __popc(m & lt)] = lk;
        pp_entries += __popc(m);
        pp_pending += (int)__reduce_add_sync(0xffffffffu, open_leaf ? lk.y : 0u);
      }
      __syncwarp();
      if (pc_pending >= 32) {
        pc_out[pc_written + lane] = ws.pcq[lane];
        pc_written += 32;
        const unsigned mv = (lane + 32 < pc_pending) ? ws.pcq[lane + 32] : 0u;
        __syncwarp();
        ws.pcq[lane] = mv;
        pc_pending -= 32;
        __syncwarp();
      }
      while (pp_pending >= 32) { flush_pp(32); pp_pending -= 32; }
    }
    if (pc_pending > 0 && lane < pc_pending) pc_out[pc_written + lane] = ws.pcq[lane];
    if (pp_pending > 0) flush_pp(pp_pending);
    __syncwarp();
  }
}

template <int TPL>
__global__ void __launch_bounds__(WALK_WARPS * 32, walk_minb(TPL)) eval_lists_kernel(const ListParams L) {
  __shared__ WarpSmem smem[WALK_WARPS];
  WarpSmem &ws = smem[threadIdx.x >> 5];
  const WalkParams &P = L.P;
  const int lane = threadIdx.x & 31;
  constexpr unsigned GS = 32u * TPL;
  for (;;) {
    unsigned item = 0;
    if (lane == 0) item = atomicAdd(L.ticket, 1u);
    item = __shfl_sync(0xffffffffu, item, 0);
    if (item >= P.n_groups) break;
    const unsigned g = L.gorder[item];
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
      float4 p = P.spos[g0 + (j < gsize ? j : gsize - 1)];
      T.x[t] = p.x; T.y[t] = p.y; T.z[t] = p.z;
      T.ax[t] = T.ay[t] = T.az[t] = T.ph[t] = T.phq[t] = 0.0f;
      if (j >= gsize) T.slot[t] = 0xffffffffu;
    }
    if constexpr (TPL == 2 && BH_PACKED) {
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
    const uint2 cnt = P.gcount[g];  // exact list lengths of the last fused pass (n_pp, n_pc)
    const uint32_t *pc_in = L.pc_list + L.pc_off[g], *pp_in = L.pp_list + L.pp_off[g];
    int unfolded = 0;
    for (unsigned base = 0; base < cnt.y; base += 32) {
      const int c = (int)min(32u, cnt.y - base);
      if (lane < c) ws.pcq[lane] = pc_in[base + lane];
      __syncwarp();
      stage_pc(ws, lane, c, P);
      eval_pc_tile<TPL>(ws, c, T, P.eps2);
      if (++unfolded >= FOLD_EVERY) { fold_tile<TPL>(T, R); unfolded = 0; }
      __syncwarp();
    }
    for (unsigned base = 0; base < cnt.x; base += 32) {
      const int c = (int)min(32u, cnt.x - base);
      unsigned pidx = 0;
      if (lane < c) { pidx = pp_in[base + lane]; ws.pp[lane] = P.spos[pidx]; ws.ppidx[lane] = pidx; }
      const bool own = __any_sync(0xffffffffu, lane < c && (pidx - (uint32_t)g0) < gsize);
      __syncwarp();
      eval_pp_tile<TPL>(ws, c, own, T, P.eps2);
      if (++unfolded >= FOLD_EVERY) { fold_tile<TPL>(T, R); unfolded = 0; }
      __syncwarp();
    }
    fold_tile<TPL>(T, R);
#pragma unroll
    for (int t = 0; t < TPL; ++t) {
      unsigned j = lane + 32u * t;
      if (j < gsize) L.out[g0 + j] = make_float4(R.get(0, t), R.get(1, t), R.get(2, t), R.get(3, t));
    }
  }
}

}  // namespace bh

extern "C" int tree_measure_listeval(tree_ctx *t, double *ms /*[2]: list walk, evaluation*/, double *max_rel) {
  using namespace bh;
  if (!t) return TREE_ERR_ARG;
  if (!ms || !max_rel) return set_err(t, TREE_ERR_ARG, "tree_measure_listeval: NULL");
  if (!t->have_force || t->group != 64 || t->shard_world > 1)
    return set_err(t, TREE_ERR_ORDER, "tree_measure_listeval needs a force pass on an unsharded context with group size 64");
  int prev_dev = -1;
  cudaGetDevice(&prev_dev);
  cudaSetDevice(t->device);
  cudaStreamSynchronize(t->stream);
  const unsigned ng = (unsigned)t->n_groups;
  std::vector<uint2> cnt(ng);
  cudaMemcpy(cnt.data(), t->b.gcount, ng * sizeof(uint2), cudaMemcpyDeviceToHost);
  std::vector<uint32_t> pc_off(ng), pp_off(ng), gorder(ng);
  unsigned long long tpc = 0, tpp = 0;
  for (unsigned g = 0; g < ng; ++g) {
    pc_off[g] = (uint32_t)tpc; pp_off[g] = (uint32_t)tpp;
    tpc += (cnt[g].y + 31u) / 32u * 32u; tpp += (cnt[g].x + 31u) / 32u * 32u;
    gorder[g] = g;
  }
  if (tpc >= (1ull << 32) || tpp >= (1ull << 32)) return set_err(t, TREE_ERR_ARG, "tree_measure_listeval: lists beyond 2^32 entries");
  std::stable_sort(gorder.begin(), gorder.end(), [&](uint32_t a, uint32_t b) {
    return 13ull * cnt[a].x + 37ull * cnt[a].y > 13ull * cnt[b].x + 37ull * cnt[b].y; });
  ListParams L;
  uint32_t *d_pc_off, *d_pp_off, *d_gorder, *d_pc, *d_pp; unsigned *d_ticket; float4 *d_out;
  if (cudaMalloc(&d_pc_off, ng * 4) || cudaMalloc(&d_pp_off, ng * 4) || cudaMalloc(&d_gorder, ng * 4) ||
      cudaMalloc(&d_pc, (tpc + 32) * 4) || cudaMalloc(&d_pp, (tpp + 32) * 4) || cudaMalloc(&d_ticket, 4) ||
      cudaMalloc(&d_out, (size_t)t->N * 16)) { cudaGetLastError(); return set_err(t, TREE_ERR_NOMEM, "tree_measure_listeval: cudaMalloc"); }
  cudaMemcpy(d_pc_off, pc_off.data(), ng * 4, cudaMemcpyHostToDevice);
  cudaMemcpy(d_pp_off, pp_off.data(), ng * 4, cudaMemcpyHostToDevice);
  cudaMemcpy(d_gorder, gorder.data(), ng * 4, cudaMemcpyHostToDevice);
  WalkParams &P = L.P;
  P.spos = t->b.spos; P.c_test = t->b.c_test; P.c_link = t->b.c_link;
  P.c_cm = t->b.c_cm; P.c_qa = t->b.c_qa; P.c_qb = t->b.c_qb;
  P.gbox = t->b.gbox; P.sacc = t->b.sacc; P.gcount = t->b.gcount; P.info = t->d_info; P.n_peers = 0;
  P.N = t->N; P.n_groups = ng; P.eps2 = t->eps * t->eps; P.svel = nullptr; P.kick_hdt = 0.f; P.reuse_mode = 0;
  P.order = nullptr; P.out_acc = nullptr; P.out_pot = nullptr; P.c_q = nullptr; P.gscale = nullptr;
  L.gorder = d_gorder; L.pc_off = d_pc_off; L.pp_off = d_pp_off; L.pc_list = d_pc; L.pp_list = d_pp; L.out = d_out;
  L.ticket = d_ticket;
  cudaEvent_t e0, e1, e2;
  cudaEventCreate(&e0); cudaEventCreate(&e1); cudaEventCreate(&e2);
  float best[2] = {1e30f, 1e30f};
  for (int rep = 0; rep < 3; ++rep) {
    cudaMemsetAsync(d_ticket, 0, 4, t->stream);
    cudaEventRecord(e0, t->stream);
    walk_lists_kernel<<<t->sm_count * COUNT_MINB, WALK_WARPS * 32, 0, t->stream>>>(L);
    cudaEventRecord(e1, t->stream);
    cudaMemsetAsync(d_ticket, 0, 4, t->stream);
    cudaEventRecord(e1, t->stream);
    eval_lists_kernel<2><<<t->sm_count * walk_minb(2), WALK_WARPS * 32, 0, t->stream>>>(L);
    cudaEventRecord(e2, t->stream);
    if (cudaStreamSynchronize(t->stream) != cudaSuccess) return set_err(t, TREE_ERR_CUDA, "tree_measure_listeval");
    t->launches += 2;
    float a = 0, b = 0;
    cudaEventElapsedTime(&a, e0, e1); cudaEventElapsedTime(&b, e1, e2);
    best[0] = std::min(best[0], a); best[1] = std::min(best[1], b);
  }
  ms[0] = best[0]; ms[1] = best[1];
  std::vector<float4> ra(t->N), rb(t->N);
  cudaMemcpy(ra.data(), t->b.sacc, (size_t)t->N * 16, cudaMemcpyDeviceToHost);
  cudaMemcpy(rb.data(), d_out, (size_t)t->N * 16, cudaMemcpyDeviceToHost);
  double worst = 0;
  for (long long i = 0; i < t->N; ++i) {
    const double dx = ra[i].x - rb[i].x, dy = ra[i].y - rb[i].y, dz = ra[i].z - rb[i].z;
    const double nn = std::sqrt((double)ra[i].x * ra[i].x + (double)ra[i].y * ra[i].y + (double)ra[i].z * ra[i].z);
    worst = std::max(worst, std::sqrt(dx * dx + dy * dy + dz * dz) / nn);
  }
  *max_rel = worst;
  cudaFree(d_pc_off); cudaFree(d_pp_off); cudaFree(d_gorder); cudaFree(d_pc); cudaFree(d_pp); cudaFree(d_ticket); cudaFree(d_out);
  cudaEventDestroy(e0); cudaEventDestroy(e1); cudaEventDestroy(e2);
  if (prev_dev >= 0) cudaSetDevice(prev_dev);
  return 0;
}
