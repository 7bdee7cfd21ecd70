// C ABI of libbhtree.so (include/tree.h): context, buffer management, call sequencing, debug
// readback. Every step of the path runs in the kernels of bh_build.cu / bh_force.cu.
#include <cstring>
#include <new>
#include <vector>

#include "bh_common.cuh"

namespace bh {

int set_err(tree_ctx *t, int code, const char *what, cudaError_t ce) {
  if (t) {
    t->err = what ? what : "";
    if (ce != cudaSuccess) { t->err += ": "; t->err += cudaGetErrorString(ce); }
  }
  return code;
}

// Errors of asynchronous passes (tree.h "asynchronous errors"), looked at after a read-back of DevInfo into t->h_info:
// each is reported once, by the first synchronising call after it happened.
int check_sticky(tree_ctx *t) {
  DevInfo *h = t->h_info;
  if (h->cells_overflow) {
    const long long need = h->cells_overflow;
    h->cells_overflow = 0;
    cudaMemsetAsync(&t->d_info->cells_overflow, 0, sizeof(unsigned), t->stream);
    t->built = false;       // the state (positions, velocities, order) is intact, the tree and the last force are not
    t->have_force = false;
    t->n_cells = need;      // the next rebuild sizes its cell arrays for it
    return set_err(t, TREE_ERR_NOMEM,
                   "tree_leapfrog: the rebuilt tree needed more cells than were allocated; the state is frozen after that "
                   "step's drift: read it with tree_get_state and call tree_build");
  }
  if (h->nonfinite_sticky) {
    h->nonfinite_sticky = 0;
    cudaMemsetAsync(&t->d_info->nonfinite_sticky, 0, sizeof(unsigned), t->stream);
    t->built = false;
    t->have_force = false;
    return set_err(t, TREE_ERR_NONFINITE, "tree_leapfrog: a position became non-finite");
  }
  if (h->walk_overflow_sticky) {
    h->walk_overflow_sticky = 0;
    cudaMemsetAsync(&t->d_info->walk_overflow_sticky, 0, sizeof(unsigned), t->stream);
    return set_err(t, TREE_ERR_CUDA, "force walk: stack overflow in a force pass since the last check, results invalid");
  }
  return 0;
}

template <typename T>
static int dev_alloc(tree_ctx *t, T *&p, long long n) {
  if (p) { cudaFree(p); p = nullptr; }
  if (n <= 0) n = 1;
  cudaError_t e = cudaMalloc((void **)&p, (size_t)n * sizeof(T));
  if (e != cudaSuccess) {
    p = nullptr;
    cudaGetLastError();
    return set_err(t, TREE_ERR_NOMEM, "cudaMalloc", e);
  }
  return 0;
}

#define BH_TRY(x) do { int _rc = (x); if (_rc) return _rc; } while (0)

// Every entry point works on the context's device and leaves the caller's current device as it found it.
struct DeviceScope {
  int prev = -1;
  cudaError_t err = cudaSuccess;
  explicit DeviceScope(int dev) {
    err = cudaGetDevice(&prev);
    if (err == cudaSuccess && prev != dev) err = cudaSetDevice(dev); else if (err == cudaSuccess) prev = -1;
  }
  ~DeviceScope() { if (prev >= 0) cudaSetDevice(prev); }
};
#define BH_DEVICE(t)                                                                        \
  bh::DeviceScope _dev_scope((t)->device);                                                  \
  if (_dev_scope.err != cudaSuccess) return bh::set_err((t), TREE_ERR_CUDA, "cudaSetDevice", _dev_scope.err)

static size_t slab_results_bytes(long long cap, long long ng) { return 2 * (size_t)cap * sizeof(float4) + 2 * (size_t)ng * sizeof(uint2); }
static size_t slab_bytes(long long cap, long long ng) {
  return slab_results_bytes(cap, ng) + (size_t)cap * sizeof(uint64_t) + (size_t)cap * sizeof(uint32_t);
}

// the exchanged sorted keys / previous slots of a sharded step inside a slab (8-byte aligned: the results are 16 N + 8 n_g)
void shard_xviews(const tree_ctx *t, void *base, uint64_t **xkey, uint32_t **xperm) {
  const long long ng = (t->cap + t->group - 1) / t->group;
  char *p = (char *)base + slab_results_bytes(t->cap, ng);
  *xkey = (uint64_t *)p;
  *xperm = (uint32_t *)(p + (size_t)t->cap * sizeof(uint64_t));
}

// result buffers inside a slab of `t`'s reserved sizes (the local one or a mapped peer's)
void shard_views(const tree_ctx *t, void *base, int parity, float4 **sacc, uint2 **gcount) {
  const long long ng = (t->cap + t->group - 1) / t->group;
  char *p = (char *)base;
  *sacc = (float4 *)(p + (size_t)parity * (size_t)t->cap * sizeof(float4));
  *gcount = (uint2 *)(p + 2 * (size_t)t->cap * sizeof(float4) + (size_t)parity * (size_t)ng * sizeof(uint2));
}

static void detach_peers(tree_ctx *t) {
  for (int r = 0; r < TREE_SHARD_MAX_WORLD; ++r) {
    if (t->peer_base[r] && t->peer_ipc[r]) cudaIpcCloseMemHandle(t->peer_base[r]);
    t->peer_base[r] = nullptr;
    t->peer_ipc[r] = false;
  }
  cudaGetLastError();
}

static int ensure_particles(tree_ctx *t, long long N) {
  if (N <= t->cap) return 0;
  if (t->shard_world > 1 && t->cap > 0)
    return set_err(t, TREE_ERR_ORDER, "sharded context: N exceeds the capacity given to tree_reserve");
  long long cap = N;
  Buffers &b = t->b;
  t->cap = 0;
  BH_TRY(dev_alloc(t, b.posm, cap));
  for (int k = 0; k < 2; ++k) {
    BH_TRY(dev_alloc(t, b.key[k], cap)); BH_TRY(dev_alloc(t, b.idx[k], cap));
    BH_TRY(dev_alloc(t, b.spos2[k], cap)); BH_TRY(dev_alloc(t, b.svel2[k], cap)); BH_TRY(dev_alloc(t, b.order2[k], cap));
  }
  t->cur = 0;
  b.spos = b.spos2[0]; b.svel = b.svel2[0]; b.order = b.order2[0];
  t->state_valid = false;
  BH_TRY(dev_alloc(t, b.lv, cap));
  long long ng = (cap + t->group - 1) / t->group;
  BH_TRY(dev_alloc(t, b.gbox, 6 * ng));
  BH_TRY(dev_alloc(t, b.gbox_prev, 6 * ng));
  t->prev_valid = false;
  {
    char *slab = (char *)b.shard_slab;
    BH_TRY(dev_alloc(t, slab, (long long)slab_bytes(cap, ng)));
    b.shard_slab = slab;
    BH_CUDA(cudaMemsetAsync(slab, 0, slab_bytes(cap, ng), t->stream));
  }
  BH_TRY(dev_alloc(t, b.gcost, ng));
  if (ng >= (1ll << 26)) return set_err(t, TREE_ERR_ARG, "too many groups (needs < 2^26)");
  t->head_cap = ng / 8 + 1024;
  t->tail_cap = 4ll * 2 * t->sm_count * 16;  // 4 parts x (2 x resident warps) groups
  const long long part_cap = t->head_cap + t->tail_cap;
  BH_TRY(dev_alloc(t, b.sched_a, ng));
  BH_TRY(dev_alloc(t, b.sched_b, ng + 2));  // also holds the 64-bit partial cost sums of the shard partition
  BH_TRY(dev_alloc(t, b.gdone, ng));
  BH_TRY(dev_alloc(t, b.gparts, ng));
  BH_TRY(dev_alloc(t, b.gthresh, ng));
  BH_TRY(dev_alloc(t, b.tasks, ng + part_cap));
  BH_TRY(dev_alloc(t, b.part, part_cap * t->group));
  BH_TRY(dev_alloc(t, b.trace, ng + part_cap));
  // scan scratch: 256 digits x sort tiles (4096 per tile) or 23 levels x tree tiles (512 per tile)
  long long s1 = 256 * ((cap + 4095) / 4096), s2 = (long long)NLEVELS * ((cap + 511) / 512);
  t->scan_cap = (s1 > s2 ? s1 : s2) + 4096;
  BH_TRY(dev_alloc(t, b.scan_tmp, t->scan_cap));
  BH_TRY(dev_alloc(t, b.scan_blk, t->scan_cap / 4096 + 16));
  BH_TRY(dev_alloc(t, b.sort_hist, 8 * 256 + 8));
  t->sort_status_cap = 256 * ((cap + 2047) / 2048);
  BH_TRY(dev_alloc(t, b.sort_status, t->sort_status_cap));
  BH_CUDA(cudaMemsetAsync(b.sort_status, 0, (size_t)t->sort_status_cap * sizeof(unsigned long long), t->stream));
  t->sort_epoch = 0;
  t->cap = cap;
  for (int k = 0; k < 2; ++k) shard_views(t, b.shard_slab, k, &b.sacc2[k], &b.gcount2[k]);
  shard_xviews(t, b.shard_slab, &b.xkey, &b.xperm);
  t->split_valid = false;
  b.sacc = b.sacc2[t->pass & 1];
  b.gcount = b.gcount2[t->pass & 1];
  t->have_vel = false;
  t->have_force = false;
  t->built = false;
  return 0;
}

int ensure_cells(tree_ctx *t, long long nc) {
  if (nc <= t->cell_cap) return 0;
  long long cap = nc + nc / 4 + 1024;
  Buffers &b = t->b;
  BH_TRY(dev_alloc(t, b.c_level, cap));
  BH_TRY(dev_alloc(t, b.c_first, cap));
  BH_TRY(dev_alloc(t, b.c_count, cap));
  BH_TRY(dev_alloc(t, b.c_fcall, cap + 1));
  BH_TRY(dev_alloc(t, b.c_link, cap));
  BH_TRY(dev_alloc(t, b.c_cm, cap));
  BH_TRY(dev_alloc(t, b.c_qa, cap));
  BH_TRY(dev_alloc(t, b.c_qb, cap));
  BH_TRY(dev_alloc(t, b.c_test, cap));
  if (t->mac == TREE_MAC_BMAX) { BH_TRY(dev_alloc(t, b.c_tlo, cap)); BH_TRY(dev_alloc(t, b.c_thi, cap)); }
  t->cell_cap = cap;
  return 0;
}

// Buffers of the relative criterion (tree_set_mac_relative), sized like the particle and cell arrays they go with.
static int ensure_relative(tree_ctx *t) {
  Buffers &b = t->b;
  if (t->rel_cap != t->cap) {
    t->rel_cap = 0;
    t->amag_valid = false;
    BH_TRY(dev_alloc(t, b.amag2[0], t->cap));
    BH_TRY(dev_alloc(t, b.amag2[1], t->cap));
    BH_TRY(dev_alloc(t, b.gscale, (t->cap + t->group - 1) / t->group));
    t->rel_cap = t->cap;
  }
  if (t->rel_cell_cap != t->cell_cap) {
    t->rel_cell_cap = 0;
    BH_TRY(dev_alloc(t, b.c_q, t->cell_cap));
    t->rel_cell_cap = t->cell_cap;
  }
  return 0;
}

static void free_all(tree_ctx *t) {
  detach_peers(t);
  Buffers &b = t->b;
  void *ptrs[] = {b.posm, b.key[0], b.key[1], b.idx[0], b.idx[1], b.spos2[0], b.spos2[1], b.svel2[0], b.svel2[1], b.order2[0], b.order2[1],
                  b.scan_tmp, b.scan_blk, b.sort_hist, b.sort_status, b.shard_slab, b.gcost,
                  b.lv, b.gbox, b.gbox_prev, b.sched_a, b.sched_b, b.gdone, b.gparts, b.gthresh, b.tasks, b.part, b.trace, b.c_level, b.c_first, b.c_count, b.c_fcall, b.c_link, b.c_cm, b.c_qa, b.c_qb,
                  b.c_test, b.c_tlo, b.c_thi, b.in_pos, b.in_mass, b.out_acc, b.out_pot, b.amag2[0], b.amag2[1], b.gscale, b.c_q};
  for (void *p : ptrs) if (p) cudaFree(p);
  b = Buffers();
}

static inline void rec(tree_ctx *t, int e) { if (t->ev_valid[e]) cudaEventRecord(t->ev[e], t->stream); }

// tree_build: the sort's payload is the caller index; the particles are gathered from the staging copy posm
static int build_from_posm(tree_ctx *t) {
  BH_TRY(run_keys(t, t->b.posm));
  rec(t, EV_KEYS);
  BH_TRY(run_sort(t));
  rec(t, EV_SORT);
  rec(t, EV_SORT2);
  BH_TRY(run_permute_build(t));
  rec(t, EV_PERM);
  t->state_valid = true;
  BH_TRY(run_tree(t, /*async=*/false));
  rec(t, EV_BUILD);
  BH_TRY(run_groups_moments(t));
  if (t->shard_world > 1) BH_TRY(run_save_splitters(t));
  rec(t, EV_MOM);
  t->built = true;
  return 0;
}

// First half of a force pass: everything up to and including the fused walk + force kernel.  The pass
// writes into the result buffers of parity (pass & 1); the other parity still holds the previous pass
// (its per-group counts schedule this one, and a sharded peer may still be reading it).
// kick_hdt != 0 (tree_leapfrog on one context): the walk's epilogue also applies the step's closing half kick.
// acc / pot (tree_force on one context): the walk's epilogue writes the results to the caller's arrays as well.
static int force_begin_impl(tree_ctx *t, float theta, float eps, float kick_hdt, float *acc = nullptr, float *pot = nullptr) {
  if (t->shard_world > 1)
    for (int r = 0; r < t->shard_world; ++r)
      if (r != t->shard_rank && !t->peer_base[r]) return set_err(t, TREE_ERR_ORDER, "sharded context: a peer is not attached");
  if (t->rel_on) {  // before the pass moves on to the other result buffer
    BH_TRY(ensure_relative(t));
    if (t->amag_valid) BH_TRY(run_group_scale(t));
  }
  t->pass++;
  t->b.sacc = t->b.sacc2[t->pass & 1];
  t->b.gcount = t->b.gcount2[t->pass & 1];
  rec(t, EV_F0);
  BH_TRY(run_opening(t, theta));
  // A force pass after a fresh tree_build normally estimates the cost of every group with a counting walk.  If the
  // previous pass on this context saw the same number of particles and nearly every group's box is where it was (the
  // caller integrates the particles itself and rebuilds every step, or asks for another theta), that pass's exact
  // counts are the better estimate, as in tree_leapfrog: no counting walk, a better-balanced task list.  The check and
  // the decision stay on the device (reuse_mode 2): no read-back.
  const int mode_in = t->reuse_mode;
  if (mode_in == 0 && t->shard_world <= 1 && t->prev_valid && t->prev_N == t->N) {
    BH_TRY(run_box_check(t));
    t->reuse_mode = 2;
  }
  const int wrc = run_walk(t, eps, kick_hdt, acc, pot);  // records EV_OPEN before and EV_WALK after the walk kernel
  t->reuse_mode = mode_in;
  if (wrc) return wrc;
  BH_CUDA(cudaMemcpyAsync(t->b.gbox_prev, t->b.gbox, (size_t)t->n_groups * 6 * sizeof(float), cudaMemcpyDeviceToDevice, t->stream));
  t->prev_valid = true;
  t->prev_N = t->N;
  t->theta = theta; t->eps = eps;
  t->have_force = false;
  t->force_open = true;
  return 0;
}

// Second half: results to the caller's arrays if it gave any (in a sharded pass, after the caller's barrier).
static int force_end_impl(tree_ctx *t, float *acc, float *pot) {
  BH_TRY(run_scatter_out(t, acc, pot));
  if (t->rel_on) {  // |a| of this pass scales the next one
    BH_TRY(run_amag_from_acc(t));
    t->amag_valid = true;
  }
  rec(t, EV_UNPERM);
  t->force_open = false;
  t->have_force = true;
  return 0;
}

static int force_impl(tree_ctx *t, float theta, float eps, float *acc, float *pot) {
  if (t->shard_world > 1) {
    BH_TRY(force_begin_impl(t, theta, eps, 0.0f));
    return force_end_impl(t, acc, pot);
  }
  BH_TRY(force_begin_impl(t, theta, eps, 0.0f, acc, pot));  // a11 fused into the walk's epilogue
  return force_end_impl(t, nullptr, nullptr);
}

// One step without a host round trip: the state stays in slot order, the cell arrays
// are used up to a bound the device checks, the cell count travels back asynchronously for the next step.
// Phase 1: kick + drift + bbox, keys, sort.  A sharded context sorts only its own key range and stores the sorted run
// into every rank (run_sort_bucket); the caller's barrier follows, then phase 2 (tree_leapfrog_mid).
static int step_phase1(tree_ctx *t, float dt) {
  // room for this step's tree: the latest known cell count plus a margin (grown here, synchronously, when the
  // margin has been used up: the arrays are rebuilt below anyway)
  poll_cells(t);
  const long long want = t->n_cells + t->n_cells / 8 + 1024;
  if (want > t->cell_cap) {
    BH_CUDA(cudaStreamSynchronize(t->stream));
    BH_TRY(ensure_cells(t, want));
  }
  if (t->shard_world > 1) {
    for (int r = 0; r < t->shard_world; ++r)
      if (r != t->shard_rank && !t->peer_base[r]) return set_err(t, TREE_ERR_ORDER, "sharded context: a peer is not attached");
    if (!t->split_valid) BH_TRY(run_save_splitters(t));  // (normally saved by the previous rebuild)
  }
  rec(t, EV_I0);
  BH_TRY(run_kick_drift_bbox(t, dt));
  rec(t, EV_I1);
  t->built = false;
  t->have_force = false;
  rec(t, EV_B0);
  BH_TRY(run_keys(t, t->b.spos));
  rec(t, EV_KEYS);
  if (t->shard_world > 1) BH_TRY(run_sort_bucket(t)); else BH_TRY(run_sort(t));
  rec(t, EV_SORT);
  t->step_open = true;
  t->step_mid_done = false;
  t->step_dt = dt;
  return 0;
}

// Phase 2: gather the state into the new order, octree, moments, first half of the force pass.
static int step_phase2(tree_ctx *t) {
  rec(t, EV_SORT2);
  BH_TRY(run_permute_step(t));
  rec(t, EV_PERM);
  BH_TRY(run_tree(t, /*async=*/true));
  rec(t, EV_BUILD);
  BH_TRY(run_groups_moments(t));
  if (t->shard_world > 1) BH_TRY(run_save_splitters(t));  // for the next step, before any peer can store new keys here
  rec(t, EV_MOM);
  t->built = true;
  t->reuse_mode = 1;  // same particles one step later: last pass's counts predict this pass's costs
  const int frc = force_begin_impl(t, t->theta, t->eps, t->shard_world <= 1 ? 0.5f * t->step_dt : 0.0f);
  t->reuse_mode = 0;
  if (frc) return frc;
  t->step_mid_done = true;
  return 0;
}

static int leapfrog_begin_impl(tree_ctx *t, float dt) {
  BH_TRY(step_phase1(t, dt));
  if (t->shard_world <= 1) BH_TRY(step_phase2(t));
  return 0;
}

static int leapfrog_end_impl(tree_ctx *t) {
  if (!t->step_mid_done) return set_err(t, TREE_ERR_ORDER, "sharded context: tree_leapfrog_mid (after the first barrier) is missing");
  BH_TRY(force_end_impl(t, nullptr, nullptr));
  rec(t, EV_I2);
  if (t->shard_world > 1) BH_TRY(run_kick(t, t->step_dt));  // one context: done in the walk's epilogue
  rec(t, EV_I3);
  t->step_open = false;
  return 0;
}

}  // namespace bh

using namespace bh;

extern "C" {

int tree_create(tree_ctx **out, int device, void *cuda_stream, int leaf_size, int group_size) {
  if (!out) return TREE_ERR_ARG;
  *out = nullptr;
  if (leaf_size < 1 || leaf_size > 32) return TREE_ERR_ARG;
  if (group_size != 32 && group_size != 64 && group_size != 128) return TREE_ERR_ARG;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) { cudaGetLastError(); return TREE_ERR_CUDA; }
  tree_ctx *t = new (std::nothrow) tree_ctx();
  if (!t) return TREE_ERR_NOMEM;
  t->device = device;
  t->stream = (cudaStream_t)cuda_stream;
  t->leaf = leaf_size;
  t->group = group_size;
  for (int i = 0; i < 24; ++i) t->ev_valid[i] = false;
  for (int i = 0; i < TREE_NPHASE; ++i) t->ms[i] = 0.0;
  DeviceScope scope(device);
  if (scope.err != cudaSuccess) { delete t; return TREE_ERR_CUDA; }
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, device) == cudaSuccess) t->sm_count = prop.multiProcessorCount;
  if (cudaMalloc((void **)&t->d_info, sizeof(DevInfo)) != cudaSuccess ||
      cudaMallocHost((void **)&t->h_info, sizeof(DevInfo)) != cudaSuccess ||
      cudaMallocHost((void **)&t->h_async, sizeof(DevInfo)) != cudaSuccess ||
      cudaEventCreateWithFlags(&t->ev_async, cudaEventDisableTiming) != cudaSuccess ||
      cudaMalloc((void **)&t->d_hlut, HLUT3_OFFSET + HLUT3_ENTRIES * sizeof(uint16_t)) != cudaSuccess) {
    cudaGetLastError();
    tree_destroy(t);
    return TREE_ERR_NOMEM;
  }
  cudaMemset(t->d_info, 0, sizeof(DevInfo));
  memset(t->h_info, 0, sizeof(DevInfo));
  memset(t->h_async, 0, sizeof(DevInfo));
  uint8_t lut[24 * 8];
  build_hilbert_lut(lut);
  cudaMemcpy(t->d_hlut, lut, sizeof(lut), cudaMemcpyHostToDevice);
  {
    std::vector<uint16_t> lut3(HLUT3_ENTRIES);
    build_hilbert_lut3(lut, lut3.data());
    cudaMemcpy(t->d_hlut + HLUT3_OFFSET, lut3.data(), HLUT3_ENTRIES * sizeof(uint16_t), cudaMemcpyHostToDevice);
  }
  for (int i = 0; i < EV_COUNT; ++i) t->ev_valid[i] = cudaEventCreate(&t->ev[i]) == cudaSuccess;
  *out = t;
  return TREE_OK;
}

int tree_destroy(tree_ctx *t) {
  if (!t) return TREE_ERR_ARG;
  DeviceScope scope(t->device);
  cudaStreamSynchronize(t->stream);
  free_all(t);
  if (t->d_info) cudaFree(t->d_info);
  if (t->h_info) cudaFreeHost(t->h_info);
  if (t->h_async) cudaFreeHost(t->h_async);
  if (t->ev_async) cudaEventDestroy(t->ev_async);
  if (t->d_hlut) cudaFree(t->d_hlut);
  for (int i = 0; i < EV_COUNT; ++i) if (t->ev_valid[i]) cudaEventDestroy(t->ev[i]);
  cudaGetLastError();
  delete t;
  return TREE_OK;
}

int tree_build(tree_ctx *t, const float *pos, const float *mass, long long N) {
  if (!t) return TREE_ERR_ARG;
  if (!pos || !mass || N <= 0 || N > 2147483647LL) return set_err(t, TREE_ERR_ARG, "tree_build: bad argument");
  BH_DEVICE(t);
  if (t->force_open || t->step_open) return set_err(t, TREE_ERR_ORDER, "tree_build inside an open force pass");
  t->built = false;
  t->have_force = false;
  t->have_vel = false;   // the slot order changes: velocities are set again after a build (tree.h)
  t->state_valid = false;
  t->amag_valid = false; // and so are the accelerations that scale the relative criterion
  BH_TRY(ensure_particles(t, N));
  t->N = N;
  t->n_groups = (N + t->group - 1) / t->group;
  rec(t, EV_B0);
  BH_TRY(run_pack_bbox(t, pos, mass));
  return build_from_posm(t);
}

int tree_force(tree_ctx *t, float theta, float eps, float *acc, float *pot) {
  if (!t) return TREE_ERR_ARG;
  if (!(theta >= 0.0f) || !(eps >= 0.0f) || !isfinite(theta) || !isfinite(eps))
    return set_err(t, TREE_ERR_ARG, "tree_force: theta and eps must be finite and >= 0");
  if (!t->built) return set_err(t, TREE_ERR_ORDER, "tree_force before tree_build");
  if (t->force_open || t->step_open) return set_err(t, TREE_ERR_ORDER, "tree_force inside an open force pass");
  if (t->shard_world > 1) return set_err(t, TREE_ERR_ORDER, "sharded context: use tree_force_begin / barrier / tree_force_end");
  BH_DEVICE(t);
  return force_impl(t, theta, eps, acc, pot);
}

static int leapfrog_check(tree_ctx *t, float dt) {
  if (!isfinite(dt)) return set_err(t, TREE_ERR_ARG, "tree_leapfrog: dt not finite");
  if (t->force_open || t->step_open) return set_err(t, TREE_ERR_ORDER, "tree_leapfrog inside an open force pass");
  if (!t->built || !t->have_force) return set_err(t, TREE_ERR_ORDER, "tree_leapfrog before tree_build + tree_force");
  if (!t->have_vel) return set_err(t, TREE_ERR_ORDER, "tree_leapfrog before tree_set_velocity");
  return 0;
}

int tree_leapfrog(tree_ctx *t, float dt) {
  if (!t) return TREE_ERR_ARG;
  BH_TRY(leapfrog_check(t, dt));
  if (t->shard_world > 1) return set_err(t, TREE_ERR_ORDER, "sharded context: use tree_leapfrog_begin / barrier / tree_leapfrog_end");
  BH_DEVICE(t);
  BH_TRY(leapfrog_begin_impl(t, dt));
  return leapfrog_end_impl(t);
}

int tree_leapfrog_begin(tree_ctx *t, float dt) {
  if (!t) return TREE_ERR_ARG;
  BH_TRY(leapfrog_check(t, dt));
  BH_DEVICE(t);
  return leapfrog_begin_impl(t, dt);
}

int tree_leapfrog_mid(tree_ctx *t) {
  if (!t) return TREE_ERR_ARG;
  if (!t->step_open) return set_err(t, TREE_ERR_ORDER, "tree_leapfrog_mid without tree_leapfrog_begin");
  if (t->step_mid_done) return TREE_OK;  // one context: tree_leapfrog_begin has done it all
  BH_DEVICE(t);
  return step_phase2(t);
}

int tree_leapfrog_end(tree_ctx *t) {
  if (!t) return TREE_ERR_ARG;
  if (!t->step_open) return set_err(t, TREE_ERR_ORDER, "tree_leapfrog_end without tree_leapfrog_begin");
  BH_DEVICE(t);
  return leapfrog_end_impl(t);
}

static int force_check(tree_ctx *t, float theta, float eps) {
  if (!(theta >= 0.0f) || !(eps >= 0.0f) || !isfinite(theta) || !isfinite(eps))
    return set_err(t, TREE_ERR_ARG, "tree_force: theta and eps must be finite and >= 0");
  if (!t->built) return set_err(t, TREE_ERR_ORDER, "tree_force before tree_build");
  if (t->force_open || t->step_open) return set_err(t, TREE_ERR_ORDER, "tree_force inside an open force pass");
  return 0;
}

int tree_force_begin(tree_ctx *t, float theta, float eps) {
  if (!t) return TREE_ERR_ARG;
  BH_TRY(force_check(t, theta, eps));
  BH_DEVICE(t);
  return force_begin_impl(t, theta, eps, 0.0f);
}

int tree_force_end(tree_ctx *t, float *acc, float *pot) {
  if (!t) return TREE_ERR_ARG;
  if (!t->force_open || t->step_open) return set_err(t, TREE_ERR_ORDER, "tree_force_end without tree_force_begin");
  BH_DEVICE(t);
  return force_end_impl(t, acc, pot);
}

int tree_reserve(tree_ctx *t, long long N) {
  if (!t) return TREE_ERR_ARG;
  if (N <= 0 || N > 2147483647LL) return set_err(t, TREE_ERR_ARG, "tree_reserve: bad N");
  BH_DEVICE(t);
  return ensure_particles(t, N);
}

int tree_shard_config(tree_ctx *t, int rank, int world) {
  if (!t) return TREE_ERR_ARG;
  if (world < 1 || world > TREE_SHARD_MAX_WORLD || rank < 0 || rank >= world)
    return set_err(t, TREE_ERR_ARG, "tree_shard_config: need 0 <= rank < world <= TREE_SHARD_MAX_WORLD");
  if (t->force_open || t->step_open) return set_err(t, TREE_ERR_ORDER, "tree_shard_config inside an open force pass");
  if (world > 1 && t->cap <= 0) return set_err(t, TREE_ERR_ORDER, "tree_shard_config before tree_reserve");
  BH_DEVICE(t);
  BH_CUDA(cudaStreamSynchronize(t->stream));
  if (world != t->shard_world || rank != t->shard_rank) detach_peers(t);
  t->shard_rank = rank;
  t->shard_world = world;
  // The result buffers are selected by the parity of `pass`, and a sharded pass stores into the SAME parity of every
  // attached context: all contexts of a world must therefore count passes alike.  Every (re)configuration restarts the
  // count, so contexts with different histories (one ran an unsharded tree_force before, one is fresh) still agree.
  t->pass = 0;
  t->b.sacc = t->b.sacc2[0];
  t->b.gcount = t->b.gcount2[0];
  t->prev_valid = false;   // the other parity no longer holds "the previous pass"
  t->have_force = false;
  t->split_valid = false;
  return TREE_OK;
}

namespace {
struct ShardBlob {  // TREE_SHARD_HANDLE_BYTES
  cudaIpcMemHandle_t ipc;
  long long cap;
  int group, device;
  char pad[TREE_SHARD_HANDLE_BYTES - sizeof(cudaIpcMemHandle_t) - sizeof(long long) - 2 * sizeof(int)];
};
static_assert(sizeof(ShardBlob) == TREE_SHARD_HANDLE_BYTES, "blob size");
}  // namespace

int tree_shard_export(tree_ctx *t, void *handle) {
  if (!t) return TREE_ERR_ARG;
  if (!handle) return set_err(t, TREE_ERR_ARG, "tree_shard_export: NULL");
  if (t->cap <= 0 || !t->b.shard_slab) return set_err(t, TREE_ERR_ORDER, "tree_shard_export before tree_reserve");
  BH_DEVICE(t);
  ShardBlob blob;
  memset(&blob, 0, sizeof(blob));
  BH_CUDA(cudaIpcGetMemHandle(&blob.ipc, t->b.shard_slab));
  blob.cap = t->cap; blob.group = t->group; blob.device = t->device;
  memcpy(handle, &blob, sizeof(blob));
  return TREE_OK;
}

static int attach_check(tree_ctx *t, int peer_rank, long long cap, int group) {
  if (t->shard_world <= 1) return set_err(t, TREE_ERR_ORDER, "tree_shard_attach before tree_shard_config");
  if (peer_rank < 0 || peer_rank >= t->shard_world || peer_rank == t->shard_rank)
    return set_err(t, TREE_ERR_ARG, "tree_shard_attach: bad peer rank");
  if (cap != t->cap || group != t->group)
    return set_err(t, TREE_ERR_ARG, "tree_shard_attach: the peer reserved a different N or group size");
  if (t->peer_base[peer_rank]) return set_err(t, TREE_ERR_ORDER, "tree_shard_attach: peer already attached");
  return 0;
}

int tree_shard_attach(tree_ctx *t, int peer_rank, const void *handle) {
  if (!t) return TREE_ERR_ARG;
  if (!handle) return set_err(t, TREE_ERR_ARG, "tree_shard_attach: NULL");
  ShardBlob blob;
  memcpy(&blob, handle, sizeof(blob));
  BH_TRY(attach_check(t, peer_rank, blob.cap, blob.group));
  BH_DEVICE(t);
  void *base = nullptr;
  BH_CUDA(cudaIpcOpenMemHandle(&base, blob.ipc, cudaIpcMemLazyEnablePeerAccess));
  t->peer_base[peer_rank] = base;
  t->peer_ipc[peer_rank] = true;
  return TREE_OK;
}

int tree_shard_attach_local(tree_ctx *t, int peer_rank, tree_ctx *peer) {
  if (!t) return TREE_ERR_ARG;
  if (!peer || peer == t || !peer->b.shard_slab) return set_err(t, TREE_ERR_ARG, "tree_shard_attach_local: bad peer");
  BH_TRY(attach_check(t, peer_rank, peer->cap, peer->group));
  BH_DEVICE(t);
  if (peer->device != t->device) {
    int can = 0;
    BH_CUDA(cudaDeviceCanAccessPeer(&can, t->device, peer->device));
    if (!can) return set_err(t, TREE_ERR_CUDA, "tree_shard_attach_local: devices are not peer-capable");
    cudaError_t e = cudaDeviceEnablePeerAccess(peer->device, 0);
    if (e != cudaSuccess && e != cudaErrorPeerAccessAlreadyEnabled) return set_err(t, TREE_ERR_CUDA, "cudaDeviceEnablePeerAccess", e);
    cudaGetLastError();
  }
  t->peer_base[peer_rank] = peer->b.shard_slab;
  t->peer_ipc[peer_rank] = false;
  return TREE_OK;
}

int tree_shard_range(tree_ctx *t, long long *g_lo, long long *g_hi, long long *s_lo, long long *s_hi) {
  if (!t) return TREE_ERR_ARG;
  if (!t->have_force && !t->force_open) return set_err(t, TREE_ERR_ORDER, "tree_shard_range before a force pass");
  BH_DEVICE(t);
  BH_CUDA(cudaMemcpyAsync(t->h_info, t->d_info, sizeof(DevInfo), cudaMemcpyDeviceToHost, t->stream));
  BH_CUDA(cudaStreamSynchronize(t->stream));
  BH_TRY(check_sticky(t));
  const long long lo = t->h_info->g_lo, hi = t->h_info->g_hi;
  if (g_lo) *g_lo = lo;
  if (g_hi) *g_hi = hi;
  if (s_lo) *s_lo = lo * t->group < t->N ? lo * t->group : t->N;
  if (s_hi) *s_hi = hi * t->group < t->N ? hi * t->group : t->N;
  return TREE_OK;
}

int tree_set_mac(tree_ctx *t, int kind) {
  if (!t) return TREE_ERR_ARG;
  if (kind != TREE_MAC_GEOMETRIC && kind != TREE_MAC_BMAX) return set_err(t, TREE_ERR_ARG, "tree_set_mac: unknown criterion");
  if (t->force_open || t->step_open) return set_err(t, TREE_ERR_ORDER, "tree_set_mac inside an open force pass");
  BH_DEVICE(t);
  t->rel_on = false;
  t->amag_valid = false;  // steps taken from here on do not carry |a| along: a later tree_set_mac_relative starts from the last pass
  if (kind != t->mac) {
    t->mac = kind;
    t->built = false;  // the tight boxes are computed with the moments: build again
    t->have_force = false;
    if (kind == TREE_MAC_BMAX && t->cell_cap > 0 && !t->b.c_tlo) {
      BH_CUDA(cudaStreamSynchronize(t->stream));
      BH_TRY(dev_alloc(t, t->b.c_tlo, t->cell_cap));
      BH_TRY(dev_alloc(t, t->b.c_thi, t->cell_cap));
    }
  }
  return TREE_OK;
}

int tree_set_mac_relative(tree_ctx *t, float alpha, const float *amag) {
  if (!t) return TREE_ERR_ARG;
  if (!(alpha >= 0.0f) || !isfinite(alpha)) return set_err(t, TREE_ERR_ARG, "tree_set_mac_relative: alpha must be finite and >= 0");
  if (t->force_open || t->step_open) return set_err(t, TREE_ERR_ORDER, "tree_set_mac_relative inside an open force pass");
  if (t->mac != TREE_MAC_GEOMETRIC) return set_err(t, TREE_ERR_ORDER, "tree_set_mac_relative: the floor is the geometric criterion (tree_set_mac)");
  if (amag && !t->built) return set_err(t, TREE_ERR_ORDER, "tree_set_mac_relative with accelerations before tree_build");
  BH_DEVICE(t);
  t->rel_on = true;
  t->rel_alpha = alpha;
  if (t->cap > 0) BH_TRY(ensure_relative(t));
  if (amag) {
    BH_TRY(run_amag_from_caller(t, amag));
    t->amag_valid = true;
  } else if (!t->amag_valid && t->built && t->have_force) {
    BH_TRY(run_amag_from_acc(t));  // the pass before this call provides the scale
    t->amag_valid = true;
  }
  return TREE_OK;
}

int tree_set_velocity(tree_ctx *t, const float *vel) {
  if (!t) return TREE_ERR_ARG;
  if (!vel) return set_err(t, TREE_ERR_ARG, "tree_set_velocity: NULL");
  if (t->N <= 0 || !t->built) return set_err(t, TREE_ERR_ORDER, "tree_set_velocity before tree_build");
  BH_DEVICE(t);
  BH_TRY(run_set_velocity(t, vel));
  t->have_vel = true;
  return TREE_OK;
}

int tree_get_state(tree_ctx *t, float *pos, float *vel, float *acc, float *pot) {
  if (!t) return TREE_ERR_ARG;
  if (t->N <= 0 || !t->state_valid) return set_err(t, TREE_ERR_ORDER, "tree_get_state before tree_build");
  if (vel && !t->have_vel) return set_err(t, TREE_ERR_ORDER, "tree_get_state: no velocities set");
  if ((acc || pot) && !t->have_force) return set_err(t, TREE_ERR_ORDER, "tree_get_state: no force computed");
  BH_DEVICE(t);
  return run_get_state(t, pos, vel, acc, pot);
}

int tree_direct(tree_ctx *t, const long long *idx, long long n, float eps, double *acc, double *pot) {
  if (!t) return TREE_ERR_ARG;
  if (!idx || !acc || !pot || n <= 0 || !(eps >= 0.0f) || !isfinite(eps))
    return set_err(t, TREE_ERR_ARG, "tree_direct: bad argument");
  if (t->N <= 0 || !t->state_valid) return set_err(t, TREE_ERR_ORDER, "tree_direct before tree_build");
  BH_DEVICE(t);
  return run_direct(t, idx, n, eps, acc, pot);
}

int tree_build_host(tree_ctx *t, const float *pos, const float *mass, long long N) {
  if (!t) return TREE_ERR_ARG;
  if (!pos || !mass || N <= 0 || N > 2147483647LL) return set_err(t, TREE_ERR_ARG, "tree_build_host: bad argument");
  BH_DEVICE(t);
  if (N > t->staging_cap) {
    t->staging_cap = 0;
    BH_TRY(dev_alloc(t, t->b.in_pos, 3 * N));
    BH_TRY(dev_alloc(t, t->b.in_mass, N));
    BH_TRY(dev_alloc(t, t->b.out_acc, 3 * N));
    BH_TRY(dev_alloc(t, t->b.out_pot, N));
    t->staging_cap = N;
  }
  BH_CUDA(cudaMemcpyAsync(t->b.in_pos, pos, (size_t)N * 12, cudaMemcpyHostToDevice, t->stream));
  BH_CUDA(cudaMemcpyAsync(t->b.in_mass, mass, (size_t)N * 4, cudaMemcpyHostToDevice, t->stream));
  return tree_build(t, t->b.in_pos, t->b.in_mass, N);
}

int tree_force_host(tree_ctx *t, float theta, float eps, float *acc, float *pot) {
  if (!t) return TREE_ERR_ARG;
  if (t->staging_cap < t->N || t->N <= 0) return set_err(t, TREE_ERR_ORDER, "tree_force_host before tree_build_host");
  int rc = tree_force(t, theta, eps, acc ? t->b.out_acc : nullptr, pot ? t->b.out_pot : nullptr);
  if (rc) return rc;
  if (acc) BH_CUDA(cudaMemcpyAsync(acc, t->b.out_acc, (size_t)t->N * 12, cudaMemcpyDeviceToHost, t->stream));
  if (pot) BH_CUDA(cudaMemcpyAsync(pot, t->b.out_pot, (size_t)t->N * 4, cudaMemcpyDeviceToHost, t->stream));
  BH_CUDA(cudaMemcpyAsync(t->h_info, t->d_info, sizeof(DevInfo), cudaMemcpyDeviceToHost, t->stream));
  BH_CUDA(cudaStreamSynchronize(t->stream));
  BH_TRY(check_sticky(t));
  return TREE_OK;
}

int tree_energy(tree_ctx *t, double *kinetic, double *potential) {
  if (!t) return TREE_ERR_ARG;
  if (!t->have_force) return set_err(t, TREE_ERR_ORDER, "tree_energy before tree_force");
  BH_DEVICE(t);
  BH_TRY(run_energy(t));
  BH_CUDA(cudaMemcpyAsync(t->h_info, t->d_info, sizeof(DevInfo), cudaMemcpyDeviceToHost, t->stream));
  BH_CUDA(cudaStreamSynchronize(t->stream));
  BH_TRY(check_sticky(t));
  if (kinetic) *kinetic = t->h_info->ekin;
  if (potential) *potential = t->h_info->epot;
  return TREE_OK;
}

static int copy_out(tree_ctx *t, void *dst, const void *src, size_t bytes) {
  BH_CUDA(cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToHost, t->stream));
  BH_CUDA(cudaStreamSynchronize(t->stream));
  return 0;
}

int tree_get_debug(tree_ctx *t, int what, void *dst, long long *count) {
  if (!t) return TREE_ERR_ARG;
  if (!count) return set_err(t, TREE_ERR_ARG, "tree_get_debug: count is NULL");
  if (!t->built) return set_err(t, TREE_ERR_ORDER, "tree_get_debug before tree_build");
  BH_DEVICE(t);
  BH_CUDA(cudaMemcpyAsync(t->h_info, t->d_info, sizeof(DevInfo), cudaMemcpyDeviceToHost, t->stream));
  BH_CUDA(cudaStreamSynchronize(t->stream));
  BH_TRY(check_sticky(t));
  t->n_cells = t->h_info->n_cells;  // exact also after an asynchronous rebuild
  const long long N = t->N, nc = t->n_cells, ng = t->n_groups;
  switch (what) {
    case TREE_DBG_KEYS: {
      *count = N;
      if (!dst) return 0;
      // keys live in slot order after the sort: scatter back through `order` on the host
      std::vector<uint64_t> sk(N);
      std::vector<uint32_t> ord(N);
      BH_TRY(copy_out(t, sk.data(), t->b.skey, N * 8));
      BH_TRY(copy_out(t, ord.data(), t->b.order, N * 4));
      uint64_t *o = (uint64_t *)dst;
      for (long long s = 0; s < N; ++s) o[ord[s]] = sk[s];
      return 0;
    }
    case TREE_DBG_ORDER: *count = N; return dst ? copy_out(t, dst, t->b.order, N * 4) : 0;
    case TREE_DBG_SORTED_KEYS: *count = N; return dst ? copy_out(t, dst, t->b.skey, N * 8) : 0;
    case TREE_DBG_SORTED_POS: *count = N; return dst ? copy_out(t, dst, t->b.spos, N * 16) : 0;
    case TREE_DBG_CELLS: {
      *count = nc;
      if (!dst) return 0;
      std::vector<uint8_t> lv(nc);
      std::vector<uint32_t> first(nc), cnt(nc);
      std::vector<uint2> link(nc);
      BH_TRY(copy_out(t, lv.data(), t->b.c_level, nc));
      BH_TRY(copy_out(t, first.data(), t->b.c_first, nc * 4));
      BH_TRY(copy_out(t, cnt.data(), t->b.c_count, nc * 4));
      BH_TRY(copy_out(t, link.data(), t->b.c_link, nc * 8));
      int32_t *o = (int32_t *)dst;
      for (long long c = 0; c < nc; ++c) {
        bool internal = link[c].y & LEAF_FLAG;
        o[5 * c] = lv[c]; o[5 * c + 1] = (int32_t)first[c]; o[5 * c + 2] = (int32_t)cnt[c];
        o[5 * c + 3] = internal ? (int32_t)link[c].x : -1;
        o[5 * c + 4] = internal ? (int32_t)(link[c].y & ~LEAF_FLAG) : 0;
      }
      return 0;
    }
    case TREE_DBG_MOMENTS: {
      *count = nc;
      if (!dst) return 0;
      std::vector<float4> cm(nc), qa(nc), qb(nc);
      BH_TRY(copy_out(t, cm.data(), t->b.c_cm, nc * 16));
      BH_TRY(copy_out(t, qa.data(), t->b.c_qa, nc * 16));
      BH_TRY(copy_out(t, qb.data(), t->b.c_qb, nc * 16));
      float *o = (float *)dst;
      for (long long c = 0; c < nc; ++c) {
        float *r = o + 11 * c;
        r[0] = cm[c].w; r[1] = cm[c].x; r[2] = cm[c].y; r[3] = cm[c].z;
        r[4] = qa[c].x; r[5] = qa[c].y; r[6] = qa[c].z; r[7] = qb[c].x; r[8] = qb[c].y; r[9] = qb[c].z;
        r[10] = qa[c].w;
      }
      return 0;
    }
    case TREE_DBG_GROUP_BOXES: *count = ng; return dst ? copy_out(t, dst, t->b.gbox, ng * 24) : 0;
    case TREE_DBG_COUNTS:
      if (!t->have_force) return set_err(t, TREE_ERR_ORDER, "counts before tree_force");
      *count = ng;
      return dst ? copy_out(t, dst, t->b.gcount, ng * 8) : 0;
    case TREE_DBG_GRID: {
      *count = 10;
      if (!dst) return 0;
      BH_TRY(copy_out(t, t->h_info, t->d_info, sizeof(DevInfo)));
      float *o = (float *)dst;
      for (int d = 0; d < 3; ++d) { o[d] = t->h_info->lo[d]; o[3 + d] = t->h_info->hi[d]; o[6 + d] = t->h_info->origin[d]; }
      o[9] = (float)t->h_info->k;
      return 0;
    }
    case TREE_DBG_ROPEN2: {
      if (!t->have_force) return set_err(t, TREE_ERR_ORDER, "ropen2 before tree_force");
      *count = nc;
      if (!dst) return 0;
      std::vector<float4> ts(nc);
      BH_TRY(copy_out(t, ts.data(), t->b.c_test, nc * 16));
      float *o = (float *)dst;
      for (long long c = 0; c < nc; ++c) o[c] = ts[c].w;
      return 0;
    }
    case TREE_DBG_TIGHT: {
      if (t->mac != TREE_MAC_BMAX) return set_err(t, TREE_ERR_ORDER, "tight boxes exist only with TREE_MAC_BMAX");
      *count = nc;
      if (!dst) return 0;
      std::vector<float4> lo(nc), hi(nc);
      BH_TRY(copy_out(t, lo.data(), t->b.c_tlo, nc * 16));
      BH_TRY(copy_out(t, hi.data(), t->b.c_thi, nc * 16));
      float *o = (float *)dst;
      for (long long c = 0; c < nc; ++c) {
        float *r = o + 7 * c;
        r[0] = lo[c].x; r[1] = lo[c].y; r[2] = lo[c].z; r[3] = hi[c].x; r[4] = hi[c].y; r[5] = hi[c].z; r[6] = lo[c].w;
      }
      return 0;
    }
    case TREE_DBG_LEVEL_OFFSETS: {
      *count = NLEVELS + 1;
      if (!dst) return 0;
      BH_TRY(copy_out(t, t->h_info, t->d_info, sizeof(DevInfo)));
      memcpy(dst, t->h_info->level_off, sizeof(int) * (NLEVELS + 1));
      return 0;
    }
    case TREE_DBG_TASK_TRACE: {
      if (!t->have_force) return set_err(t, TREE_ERR_ORDER, "task trace before tree_force");
      BH_TRY(copy_out(t, t->h_info, t->d_info, sizeof(DevInfo)));
      *count = t->h_info->n_tasks;
      return dst ? copy_out(t, dst, t->b.trace, (size_t)t->h_info->n_tasks * 16) : 0;
    }
    default: return set_err(t, TREE_ERR_ARG, "tree_get_debug: unknown selector");
  }
}

int tree_get_stats(tree_ctx *t, double *ms, unsigned long long *n_pp, unsigned long long *n_pc) {
  if (!t) return TREE_ERR_ARG;
  BH_DEVICE(t);
  BH_CUDA(cudaStreamSynchronize(t->stream));
  auto el = [&](int a, int b) -> double {
    if (!t->ev_valid[a] || !t->ev_valid[b]) return 0.0;
    if (cudaEventQuery(t->ev[a]) != cudaSuccess || cudaEventQuery(t->ev[b]) != cudaSuccess) { cudaGetLastError(); return 0.0; }
    float f = 0.f;
    if (cudaEventElapsedTime(&f, t->ev[a], t->ev[b]) != cudaSuccess) { cudaGetLastError(); return 0.0; }
    return f > 0.f ? (double)f : 0.0;
  };
  double *m = t->ms;
  m[TREE_PH_KEYS] = el(EV_B0, EV_KEYS);
  m[TREE_PH_SORT] = el(EV_KEYS, EV_SORT);
  m[TREE_PH_PERMUTE] = el(EV_SORT2, EV_PERM);
  m[TREE_PH_BUILD] = el(EV_PERM, EV_BUILD);
  m[TREE_PH_MOMENTS] = el(EV_BUILD, EV_MOM);
  m[TREE_PH_OPENING] = t->have_force ? el(EV_F0, EV_OPEN) : 0.0;
  m[TREE_PH_SCHED] = t->have_force ? el(EV_OPEN, EV_SCHED) : 0.0;
  m[TREE_PH_WALK] = t->have_force ? el(EV_SCHED, EV_WALK) : 0.0;
  m[TREE_PH_UNPERMUTE] = t->have_force ? el(EV_WALK, EV_UNPERM) : 0.0;
  m[TREE_PH_INTEGRATE] = el(EV_I0, EV_I1) + el(EV_I2, EV_I3);
  m[TREE_PH_TOTAL] = 0.0;
  for (int i = 0; i < TREE_PH_TOTAL; ++i) m[TREE_PH_TOTAL] += m[i];
  if (ms) memcpy(ms, m, sizeof(double) * TREE_NPHASE);
  if (n_pp || n_pc) {
    BH_CUDA(cudaMemcpy(t->h_info, t->d_info, sizeof(DevInfo), cudaMemcpyDeviceToHost));
    if (n_pp) *n_pp = t->h_info->n_pp;
    if (n_pc) *n_pc = t->h_info->n_pc;
    BH_TRY(check_sticky(t));
  }
  return TREE_OK;
}

int tree_fp32_peak(tree_ctx *t, double *tflops) {
  if (!t) return TREE_ERR_ARG;
  if (!tflops) return set_err(t, TREE_ERR_ARG, "tree_fp32_peak: NULL");
  BH_DEVICE(t);
  return run_fp32_peak(t, tflops);
}

long long tree_launch_count(const tree_ctx *t) { return t ? t->launches : 0; }

const char *tree_last_error(const tree_ctx *t) { return t ? t->err.c_str() : ""; }

}  // extern "C"
