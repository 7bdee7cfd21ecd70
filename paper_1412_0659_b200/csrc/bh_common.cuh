// Shared declarations of the CUDA Barnes-Hut library (sm_100a). Product code: nothing here is
// shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <cstdint>
#include <cstdio>
#include <string>

#include "../../include/tree.h"

namespace bh {

constexpr int KEY_BITS = 21;      // bits per dimension -> 63-bit Peano-Hilbert key (S8)
constexpr int MAX_LEVEL = KEY_BITS;
constexpr int NLEVELS = MAX_LEVEL + 2;  // levels 0..21 exist; level 22 is an always-empty sentinel
constexpr uint32_t LEAF_FLAG = 0x80000000u;
constexpr int HLUT3_ENTRIES = 24 * 512;  // Hilbert table over three levels per look-up (keys_kernel), uint16 each
constexpr int HLUT3_OFFSET = 256;        // its byte offset inside tree_ctx::d_hlut (the 24 x 8 table comes first)

// Device-resident scalars of one build.
struct DevInfo {
  int lo_enc[3], hi_enc[3];  // order-preserving integer encodings of the bbox (atomicMin/Max)
  int nonfinite;             // set if a non-finite position or mass was seen
  int k;                     // cube side S = 2^k
  float lo[3], hi[3], origin[3];
  float inv;                 // 2^(21-k): grid cells per unit length
  int level_off[NLEVELS + 1];  // first BFS cell id of each level, then n_cells
  unsigned long long n_pp, n_pc;  // interaction totals of the last force pass
  unsigned long long t0_ns;       // globaltimer at the start of the last force pass (task trace origin)
  unsigned long long sched_cost;  // sum of the per-group cost estimates of the counting walk
  unsigned int group_ticket;      // dynamic group fetch counter of the counting walk
  unsigned int task_ticket;       // dynamic task fetch counter of the force walk
  unsigned int n_tasks, n_tasks_a;  // tasks in the list; of which parts of expensive groups (listed first)
  unsigned int tail_start;          // first task of the tail region (last groups, split into small tasks)
  unsigned int walk_overflow;       // set if a warp's walk stack would have overflowed (results invalid)
  unsigned int walk_overflow_sticky;  // the same, but cleared only when a synchronising call has reported it
  unsigned int sched_tot[2];      // totals of the two scheduling scans
  unsigned int g_lo, g_hi;        // groups this context walks in the current force pass (all of them unless sharded)
  double ekin, epot;
  unsigned int moved_groups;      // groups whose box is not where the previous force pass saw it (box_moved_kernel)
  unsigned int reuse_costs;       // this pass schedules by the previous pass's per-group counts (decided on the device)
  int n_cells;                    // cells of the current tree (= level_off[NLEVELS])
  int ltop;                       // levels 0..ltop hold so few cells that one block computes their moments
  unsigned int nonfinite_sticky;  // sticky: a rebuild saw a non-finite position or mass (asynchronous steps report it late)
  // sharded step (DESIGN.md §7 "partitioned sort"): key splitters of the previous sorted order and the bucket sizes
  unsigned long long split[TREE_SHARD_MAX_WORLD];   // split[r] = first key of bucket r (split[0] unused: bucket 0 starts at 0)
  unsigned int bucket_cnt[TREE_SHARD_MAX_WORLD];    // particles whose new key falls into bucket r
  unsigned int bucket_fill;                         // compaction cursor of this context's own bucket
  unsigned int cells_overflow;    // sticky: an asynchronous rebuild needed more cells than allocated; the cell count it
                                  // needed.  Every later kernel of the step pipeline does nothing while it is set.
};

struct Buffers {
  // caller order: only the staging copy of tree_build's input (x,y,z,m)
  float4 *posm = nullptr;
  // sort: key and payload, double-buffered.  Payload = caller index (tree_build) or previous slot (tree_leapfrog)
  uint64_t *key[2] = {nullptr, nullptr};
  uint32_t *idx[2] = {nullptr, nullptr};
  uint32_t *scan_tmp = nullptr;  // tile level counts of the tree build / scheduling scans (scanned in place)
  uint32_t *sort_hist = nullptr;              // [8][256] digit histograms -> global digit offsets, then 8 tile tickets
  unsigned long long *sort_status = nullptr;  // [sort tiles][256] decoupled look-back words of the one-sweep sort
  uint32_t *scan_blk = nullptr;  // block sums for the device-wide scan
  // slot (sorted) order: the STATE.  It stays in the slot order of the last sort; a leapfrog step gathers it into the
  // new order (a nearly sequential gather: few particles change their place on the curve in one step), so no array
  // is kept in caller order and results are scattered to caller order only when the caller asks for them.
  float4 *spos2[2] = {nullptr, nullptr}, *svel2[2] = {nullptr, nullptr};
  uint32_t *order2[2] = {nullptr, nullptr};
  float4 *spos = nullptr;      // = spos2[cur]: x,y,z,m
  float4 *svel = nullptr;      // = svel2[cur]: vx,vy,vz,0
  uint32_t *order = nullptr;   // = order2[cur]: order[s] = caller index of the particle in slot s
  void *shard_slab = nullptr;  // one allocation (one IPC handle): sacc2[0] | sacc2[1] | gcount2[0] | gcount2[1] | xkey | xperm
  uint64_t *xkey = nullptr;    // sharded step: the sorted keys, every rank's bucket stored at its offset by its owner
  uint32_t *xperm = nullptr;   //               and the previous slot of each sorted particle
  const uint64_t *skey = nullptr;   // the sorted keys of the current tree: key[sorted], or xkey after a sharded step
  const uint32_t *sperm = nullptr;  // payload of the last sort: idx[sorted] or xperm
  float4 *sacc2[2] = {nullptr, nullptr};  // results in slot order, double-buffered by force pass
  float4 *sacc = nullptr;                 // = sacc2[pass & 1], the buffer of the current / last force pass
  uint16_t *lv = nullptr;   // per slot: L0 | Lleaf << 5
  // groups
  float *gbox = nullptr;    // [n_groups][6]
  float *gbox_prev = nullptr;  // the group boxes of the previous force pass (is this build the same particles, moved a little?)
  uint2 *gcount2[2] = {nullptr, nullptr};  // [n_groups] n_pp, n_pc, double-buffered like sacc2
  uint2 *gcount = nullptr;                 // = gcount2[pass & 1]
  double *gcost = nullptr;  // [n_groups] cost estimate of the current pass (task list and shard partition)
  // scheduling of the force walk
  uint32_t *sched_a = nullptr, *sched_b = nullptr;  // [n_groups] part counts -> offsets (scanned in place)
  uint32_t *gdone = nullptr;   // [n_groups]
  uint8_t *gparts = nullptr;   // [n_groups]
  uint32_t *gthresh = nullptr; // [n_groups]
  uint32_t *tasks = nullptr;   // [n_groups + part_cap]
  float4 *part = nullptr;      // [part_cap][group]
  uint4 *trace = nullptr;      // [n_groups + part_cap] per-task trace of the last force pass
  // cells (BFS order)
  uint8_t *c_level = nullptr;
  uint32_t *c_first = nullptr, *c_count = nullptr, *c_fcall = nullptr;
  uint2 *c_link = nullptr;    // leaf: (first, count); internal: (first_child, n_child | LEAF_FLAG.. see bh_build.cu)
  float4 *c_cm = nullptr;     // cx,cy,cz,M
  float4 *c_qa = nullptr;     // Qxx,Qyy,Qzz,delta
  float4 *c_qb = nullptr;     // Qxy,Qxz,Qyz,tr(Q)
  float4 *c_test = nullptr;   // cx,cy,cz,r_open^2 (per force call)
  float4 *c_tlo = nullptr, *c_thi = nullptr;  // TREE_MAC_BMAX only: tight box lo x,y,z | b  and  hi x,y,z | -
  // tree_set_mac_relative only: |a| of the last force pass per slot (part of the state: gathered with it by a step),
  // alpha * min |a| per group, M l^3 per cell (per force call)
  float *amag2[2] = {nullptr, nullptr}, *gscale = nullptr, *c_q = nullptr;
  // host-call staging
  float *in_pos = nullptr, *in_mass = nullptr, *out_acc = nullptr, *out_pot = nullptr;
};

}  // namespace bh

struct tree_ctx {
  int device = 0;
  cudaStream_t stream = nullptr;
  int leaf = 16, group = 64;
  int mac = TREE_MAC_GEOMETRIC;      // acceptance criterion (tree_set_mac)
  bool rel_on = false;               // tree_set_mac_relative: the error-targeted condition on top of the geometric one
  float rel_alpha = 0.f;
  bool amag_valid = false;           // b.amag2[cur] holds |a| of every particle of the current slot order
  long long rel_cap = 0, rel_cell_cap = 0;  // capacities b.amag2 / b.gscale and b.c_q were allocated for
  long long N = 0, cap = 0;          // particles, particle capacity
  long long n_cells = 0, cell_cap = 0;  // n_cells: exact after tree_build; after an asynchronous rebuild (tree_leapfrog) the
                                        // latest count read back so far (poll_cells)
  long long cells_bound = 0;            // cells the kernels of the current tree may use / launch for (<= cell_cap)
  int cur = 0;                          // which of the state double buffers (spos2, svel2, order2) is current
  bh::DevInfo *h_async = nullptr;       // pinned: DevInfo copied back after the tree kernels of an asynchronous rebuild
  cudaEvent_t ev_async = nullptr;
  bool async_pending = false;
  long long n_groups = 0;
  long long scan_cap = 0;
  long long sort_status_cap = 0;     // words in b.sort_status
  unsigned long long sort_epoch = 0; // look-back epoch: one per sort pass, never reused before a clear
  long long head_cap = 0, tail_cap = 0;  // partial-sum slots for expensive-group parts / tail parts
  bool sort_attr_set = false;        // the sort kernel's shared-memory attributes are set on this context's device
  int sorted = 0;                    // which of key[]/idx[] holds the sorted result
  bool built = false, have_vel = false, have_force = false;
  bool state_valid = false;          // spos / svel / order hold one consistent particle set (tree_get_state, tree_direct)
  long long staging_cap = 0;         // capacity of the host-call staging buffers
  float theta = 0.f, eps = 0.f;
  int reuse_mode = 0;                // scheduling of the next force pass: 0 = counting walk, 1 = by the previous pass's
                                     // per-group counts (tree_leapfrog), 2 = decided on the device by box_moved_kernel
  bool prev_valid = false;           // b.gbox_prev and the other parity's gcount describe a finished pass over prev_N particles
  long long prev_N = 0;
  // sharded force pass: this context walks one contiguous cost-balanced range of groups and
  // stores the results into every attached context's result buffers
  int shard_rank = 0, shard_world = 1;
  unsigned pass = 0;                 // force passes begun; parity selects the result buffers
  bool force_open = false;           // between tree_force_begin and tree_force_end
  bool step_open = false;            // between tree_leapfrog_begin and tree_leapfrog_end
  bool step_mid_done = false;        // sharded step: tree_leapfrog_mid has run (begin | barrier | mid | barrier | end)
  bool slot_of_valid = false;        // the inverse of `order` (caller index -> slot) is in the spare key buffer
  bool split_valid = false;          // d_info->split holds the splitters of the current sorted order
  float step_dt = 0.f;
  float *open_acc = nullptr, *open_pot = nullptr;
  void *peer_base[TREE_SHARD_MAX_WORLD] = {};   // mapped result slab of each attached peer (nullptr: not attached)
  bool peer_ipc[TREE_SHARD_MAX_WORLD] = {};     // mapping came from cudaIpcOpenMemHandle (to be closed)
  int sm_count = 148;
  bh::Buffers b;
  bh::DevInfo *d_info = nullptr;
  bh::DevInfo *h_info = nullptr;     // pinned
  uint8_t *d_hlut = nullptr;         // Hilbert state tables (device copy): 24 x 8 bytes | at HLUT3_OFFSET: 24 x 512 uint16
  cudaEvent_t ev[24];
  bool ev_valid[24];
  double ms[TREE_NPHASE];
  long long launches = 0;
  std::string err;
};

namespace bh {

// event slots
enum { EV_B0 = 0, EV_KEYS, EV_SORT, EV_SORT2, EV_PERM, EV_BUILD, EV_MOM, EV_F0, EV_OPEN, EV_SCHED, EV_WALK, EV_UNPERM,
       EV_I0, EV_I1, EV_I2, EV_I3, EV_COUNT };

int set_err(tree_ctx *t, int code, const char *what, cudaError_t ce = cudaSuccess);
// After a read-back of DevInfo into t->h_info: report (once) a walk-stack overflow of any force pass since the last report.
int check_sticky(tree_ctx *t);

#define BH_CUDA(call)                                                      \
  do {                                                                     \
    cudaError_t _e = (call);                                               \
    if (_e != cudaSuccess) return bh::set_err(t, TREE_ERR_CUDA, #call, _e); \
  } while (0)

#define BH_LAUNCH_CHECK(name)                                                   \
  do {                                                                          \
    cudaError_t _e = cudaGetLastError();                                        \
    if (_e != cudaSuccess) return bh::set_err(t, TREE_ERR_CUDA, name, _e);      \
    t->launches++;                                                              \
  } while (0)

// phases implemented in bh_build.cu / bh_force.cu (host launchers; all enqueue on t->stream)
int run_pack_bbox(tree_ctx *t, const float *pos, const float *mass);  // caller arrays -> posm + bbox
int run_kick_drift_bbox(tree_ctx *t, float dt);                        // leapfrog: kick + drift of the slot-order state + bbox
int run_keys(tree_ctx *t, const float4 *xyzm);                         // grid + keys of posm (build) or spos (leapfrog)
int run_sort(tree_ctx *t);                            // all N keys of key[0], payload = identity
int run_sort_bucket(tree_ctx *t);                     // sharded step: count, compact and sort this context's key range, store it to all
int run_save_splitters(tree_ctx *t);                  // keys at the slot boundaries N r / world of the current sorted order
void shard_xviews(const tree_ctx *t, void *base, uint64_t **xkey, uint32_t **xperm);
int run_permute_build(tree_ctx *t);   // tree_build: posm -> spos, order (payload of the sort = caller index)
int run_permute_step(tree_ctx *t);    // tree_leapfrog: spos, svel, order -> the new slot order (payload = previous slot)
int run_tree(tree_ctx *t, bool async);  // octree construction; !async: synchronises once and sizes the cell arrays
int run_groups_moments(tree_ctx *t);
int run_opening(tree_ctx *t, float theta);
int run_amag_from_acc(tree_ctx *t);                      // relative criterion: amag[s] = |a| of the last force pass
int run_amag_from_caller(tree_ctx *t, const float *amag);  // ... or the caller's values (caller order) into slot order
int run_group_scale(tree_ctx *t);                        // gscale[g] = alpha * min amag over the group's slots
// kick_hdt != 0: v += a * kick_hdt in the walk's epilogue; out_acc / out_pot (one context): results also to the caller's arrays there
int run_walk(tree_ctx *t, float eps, float kick_hdt, float *out_acc, float *out_pot);
int run_box_check(tree_ctx *t);  // device-side: are the group boxes where the previous force pass saw them?
void shard_views(const tree_ctx *t, void *base, int parity, float4 **sacc, uint2 **gcount);
int run_scatter_out(tree_ctx *t, float *acc, float *pot);  // results to the caller's arrays (caller order)
int run_kick(tree_ctx *t, float dt);
void poll_cells(tree_ctx *t);  // non-blocking: take over the cell count of the last asynchronous rebuild if it has arrived
int run_energy(tree_ctx *t);
int run_set_velocity(tree_ctx *t, const float *vel);
int run_get_state(tree_ctx *t, float *pos, float *vel, float *acc, float *pot);
int run_direct(tree_ctx *t, const long long *idx, long long n, float eps, double *acc, double *pot);
int run_fp32_peak(tree_ctx *t, double *tflops);
int ensure_cells(tree_ctx *t, long long n_cells);
void build_hilbert_lut(uint8_t out[24 * 8]);
void build_hilbert_lut3(const uint8_t lut[24 * 8], uint16_t out[HLUT3_ENTRIES]);
int device_excl_scan(tree_ctx *t, uint32_t *a, long long n, uint32_t *total_out);

}  // namespace bh
