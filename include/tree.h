/* tree.h — C ABI of the B200-native Barnes-Hut force library (libbhtree.so).
 *
 * What it computes (arxiv 1412.0659, Bedorf et al. 2014, cited as PAPER.md:L<line>):
 * for N point masses with FP32 positions r_j and masses m_j, the
 * acceleration a_i and potential phi_i "which we collectively call the force" (L184) by the
 * Barnes-Hut tree algorithm (L31): Peano-Hilbert keys over the bounding box (L97), sort (Table
 * II L244), sparse octree with at most `leaf_size` particles per leaf (L31, L246), multipole
 * moments mass / centre of mass / quadrupole per cell (L65, L190, L247), then a fused tree-walk +
 * force pass (L67-79, L248) that evaluates particle-particle (23 flop) and particle-cell (65 flop)
 * interactions, Eqs. (1),(2) (L186-192), with Plummer softening eps and opening angle theta
 * (L31, L133), and a 2nd-order leapfrog (L121).  G = 1.  Every reading of a point PAPER.md leaves
 * open is listed in DESIGN.md ("Readings").
 *
 * Conventions
 *  - Plain C, no exceptions, never exits.  Every call returns 0 on success or a negative code:
 *      TREE_ERR_ARG      -1  bad argument (NULL, N <= 0, N > 2^31-1, theta < 0, eps < 0, NaN ...)
 *      TREE_ERR_NOMEM    -2  out of device (or pinned host) memory
 *      TREE_ERR_CUDA     -3  CUDA error; text via tree_last_error()
 *      TREE_ERR_ORDER    -4  call order (force before build, leapfrog before force/velocities)
 *      TREE_ERR_NONFINITE -5 non-finite position or mass detected while building
 *  - Pointers marked DEV are device pointers on the context's device, allocated and owned by the
 *    caller (e.g. torch tensors); pointers marked HOST are host pointers (pinned memory makes the
 *    copies faster, pageable works).  The library copies what it needs during the call and never
 *    keeps a caller pointer.  Its own buffers grow to the largest N seen and are reused.
 *  - All work is enqueued on the stream given to tree_create (NULL = the legacy default stream).
 *    tree_build synchronises that stream once (it reads the cell count back to size the cell
 *    arrays); tree_force and tree_leapfrog return after enqueueing and never wait for the device
 *    (tree_leapfrog's rebuild uses the cell arrays up to a bound the device checks, and the cell count
 *    travels back asynchronously for the next step); the *_host variants, tree_get_debug,
 *    tree_get_stats, tree_energy and tree_shard_range synchronise.
 *  - Asynchronous errors.  What an asynchronous tree_leapfrog can run into on the device is reported
 *    ONCE, by the next call that synchronises (tree_build, tree_force_host, tree_get_debug,
 *    tree_get_stats, tree_energy, tree_shard_range), however many steps were enqueued in between:
 *      TREE_ERR_NOMEM     the rebuilt tree needed more cells than allocated (the allocation follows the
 *                         last known cell count + 1/8 + 1024; the count moves by a fraction of a per
 *                         cent per step).  From that step on the device does nothing: the state
 *                         (positions after that step's drift, velocities after its first half kick) is
 *                         frozen and can be read with tree_get_state; continue with tree_build.
 *      TREE_ERR_NONFINITE a position became non-finite.
 *      TREE_ERR_CUDA      the force walk's stack guard fired (see below).
 *  - The library keeps its state (positions, velocities, forces) in the order of the last sort
 *    ("slot order") and moves it into the next order inside tree_leapfrog; the caller's order is
 *    restored only where a call hands arrays back (tree_force's acc / pot, tree_get_state).
 *  - Every call works on the context's device and restores the caller's current CUDA device before it returns.
 *  - The force walk keeps its stack in shared memory behind a guard (the bound is 32 entries per
 *    level); should the guard ever fire, the results of that pass are invalid and the NEXT call that synchronises
 *    (tree_build, tree_leapfrog's rebuild, tree_force_host, tree_energy, tree_get_stats, tree_shard_range) returns
 *    TREE_ERR_CUDA once ("stack overflow"), however many asynchronous passes were enqueued in between.
 *  - "Caller order" is the particle order of the arrays given to tree_build.  Outputs are always
 *    in caller order.  Masses must be > 0.  No two particles may share a position unless eps > 0
 *    (the self term is skipped by index, "N-1 interactions").
 */
#ifndef BHTREE_TREE_H
#define BHTREE_TREE_H

#ifdef __cplusplus
extern "C" {
#endif

#define TREE_OK 0
#define TREE_ERR_ARG (-1)
#define TREE_ERR_NOMEM (-2)
#define TREE_ERR_CUDA (-3)
#define TREE_ERR_ORDER (-4)
#define TREE_ERR_NONFINITE (-5)

typedef struct tree_ctx tree_ctx; /* opaque; owned by the library */

/* Create a context on CUDA device `device`, working on `cuda_stream` (a cudaStream_t, may be
 * NULL).  leaf_size: a cell with at most this many particles is a leaf ("we use
 * 16"); 1..32.  group_size: number of consecutive Peano-Hilbert-sorted particles that share one
 * tree walk (one warp); 32, 64 or 128 (the paper's unnamed warp-shared lists, L79). */
int tree_create(tree_ctx **out, int device, void *cuda_stream, int leaf_size, int group_size);

/* Build the tree for N particles: bounding box and PH keys, sort (L244), octree
 * (L31, L246), groups, multipole moments level by level (L65, L190, L247).
 * pos: DEV float[N][3] row-major; mass: DEV float[N].  1 <= N <= 2^31-1. */
int tree_build(tree_ctx *t, const float *pos, const float *mass, long long N);

/* Force pass on the last built tree (Eqs. (1),(2) L186-188): opening radii for
 * this theta, fused walk + evaluation, results to caller order.
 * Accuracy against the FP64 sum of the same interaction lists: |phi - phi_exact| <= 1e-5 |phi|
 * and |a - a_exact| <= max(1e-5 |a|, 2.5e-7 A), A = sum of the magnitudes of the terms of the particle's list; the
 * second term only decides where the net force cancels to less than 1/40 of that sum.
 * theta >= 0 (0 = open everything = direct summation, L31); eps >= 0 (Plummer softening).
 * acc: DEV float[N][3] or NULL; pot: DEV float[N] or NULL.  The result is also kept inside the
 * context for tree_leapfrog / tree_get_state.
 * Scheduling (results do not depend on it beyond the rounding of partial sums of split groups): the cost of every
 * group comes from a counting walk, or, when the previous pass on this context saw the same N and the group
 * boxes have hardly moved (checked on the device; one 4-byte read-back and stream synchronise), from that pass's
 * exact per-group counts. */
int tree_force(tree_ctx *t, float theta, float eps, float *acc, float *pot);

/* One kick-drift-kick step of size dt: v += a dt/2; x += v dt; rebuild the tree;
 * force with the theta, eps of the last tree_force; v += a dt/2.  Needs tree_set_velocity and
 * one tree_force before.  dt may be negative. */
int tree_leapfrog(tree_ctx *t, float dt);

int tree_destroy(tree_ctx *t);

/* ---- auxiliary ------------------------------------------------------------------------ */

/* Acceptance criterion of the walk (PAPER.md L31 names only "a multipole acceptance criterion
 * parameterized by an opening angle theta" and L133 fixes theta = 0.4 for accuracy, cost ~ theta^-3):
 *   TREE_MAC_GEOMETRIC (default; S5)  accept iff D > l / theta + delta, l = side of the cell's octant,
 *                                               delta = |centre of mass - centre of the octant|
 *   TREE_MAC_BMAX                               accept iff D > b / theta, b = distance from the cell's centre of mass to
 *                                               the farthest corner of the TIGHT bounding box of its particles (the
 *                                               bounding-radius criterion of Salmon & Warren)
 * D = distance from the group's bounding box to the cell's centre of mass in both.  Call before tree_build (the tight
 * boxes are computed with the moments); a context that is already built must be built again. */
#define TREE_MAC_GEOMETRIC 0
#define TREE_MAC_BMAX 1
int tree_set_mac(tree_ctx *t, int kind);

/* Error-targeted acceptance per group (SURVEY.md 8(f) NEXT-2 "per-group theta chosen to hit a force-error target"; not in
 * PAPER.md, which fixes theta = 0.4 "for accuracy", L133).  On top of TREE_MAC_GEOMETRIC -- which stays necessary, with the
 * theta of tree_force as a floor (theta = 1 is a sensible one) -- group g accepts cell c only if
 *     D^5 alpha a_g > M l^3,
 * a_g = the smallest |a| among the group's particles in the previous force pass on this context: the first multipole
 * term the evaluation leaves out, ~ M l^3 / D^5, stays below alpha times the group's own acceleration.  FP32, one IEEE
 * operation each: gscale = alpha * a_g; sqrt(D2) * D2 * D2 * gscale > M * l * l * l.
 *   alpha : >= 0 (0 opens everything).  Measured (profiles/r2_mac_sweep_*.md): the median error of theta = 0.4 in 0.44 x the
 *           time on the Milky-Way-shaped model, with a smaller 99th percentile; alpha = 3e-4 is better than theta = 0.4 in
 *           every error figure at about half the time.
 *   amag  : DEV float[N], caller order, |a| of every particle, or NULL.  NULL: the library uses the accelerations of its
 *           own last force pass; they travel with the particles through tree_leapfrog.  A pass with no accelerations to go
 *           by (the first one after tree_build) uses the geometric criterion alone with its theta, so the usual sequence is
 *           tree_build, tree_force(0.4, ...), tree_set_mac_relative(alpha, NULL), tree_force(1.0, ...), tree_leapfrog ...
 *           Non-NULL (needs a built tree): these values scale the next pass instead (tests: the same input to the oracle).
 * A group one of whose particles has |a| = 0 opens every cell (direct summation for that group): for systems whose net forces
 * cancel by symmetry (lattices, uniform boxes) use the geometric criterion.
 * tree_set_mac(t, kind) switches it off again.  Needs no rebuild.  Sharded contexts: every rank makes the same call at the
 * same point of the sequence (every rank holds the complete results of every pass, so all ranks derive the same scales and
 * the same lists; nothing more is communicated).  Allocates 8 bytes per particle and 4 per cell on first use. */
int tree_set_mac_relative(tree_ctx *t, float alpha, const float *amag);

/* vel: DEV float[N][3], caller order, N of the last tree_build.  tree_build forgets the velocities (it re-orders the
 * state): set them after every tree_build that is followed by tree_leapfrog. */
int tree_set_velocity(tree_ctx *t, const float *vel);

/* Current state in caller order; any pointer may be NULL.  pos, vel, acc: DEV float[N][3];
 * pot: DEV float[N]. */
int tree_get_state(tree_ctx *t, float *pos, float *vel, float *acc, float *pot);

/* Same as tree_build / tree_force with HOST buffers: the host<->device copies are part of the
 * call (this is the end-to-end path bench.py times).  tree_force_host returns after the results
 * are in acc / pot. */
int tree_build_host(tree_ctx *t, const float *pos, const float *mass, long long N);
int tree_force_host(tree_ctx *t, float theta, float eps, float *acc, float *pot);

/* Kinetic energy sum 1/2 m v^2 and potential energy 1/2 sum m phi of the current state, FP64
 * sums, written to HOST doubles (either may be NULL).  Synchronises. */
int tree_energy(tree_ctx *t, double *kinetic, double *potential);

/* Exact softened sum over ALL N particles of the current state for a list of targets (PAPER.md L29
 * "each of the N objects exerts N-1 interactions"; L184-190 with Q = 0): for target i = idx[k],
 * over all j != i (by index): phi = -sum m_j / s, a = sum m_j r / s^3, r = x_j - x_i,
 * s^2 = |r|^2 + eps^2, evaluated and accumulated in FP64 from the FP32 state.  This is the
 * "direct summation" the tree force is measured against (theta -> 0 limit, L31); it is O(n N).
 * idx: DEV int64[n], caller-order particle indices in [0, N); acc: DEV double[n][3];
 * pot: DEV double[n]; both are overwritten.  Needs tree_build (any later tree_leapfrog state is
 * the one summed).  Asynchronous on the context's stream. */
int tree_direct(tree_ctx *t, const long long *idx, long long n, float eps, double *acc, double *pot);

/* Internal arrays for the parity tests, copied to HOST memory `dst`.  *count receives the number
 * of records; with dst == NULL only *count is written.  Synchronises.  `what`: */
#define TREE_DBG_KEYS 0        /* uint64[N]     PH key per particle, caller order                  */
#define TREE_DBG_ORDER 1       /* uint32[N]     order[s] = caller index of the particle in slot s  */
#define TREE_DBG_SORTED_KEYS 2 /* uint64[N]     keys in slot order                                 */
#define TREE_DBG_CELLS 3       /* int32[n_cells][5] level, first, count, first_child(-1 leaf), n_child; BFS order */
#define TREE_DBG_MOMENTS 4     /* float[n_cells][11] M, cx,cy,cz, Qxx,Qyy,Qzz,Qxy,Qxz,Qyz, delta    */
#define TREE_DBG_GROUP_BOXES 5 /* float[n_groups][6] min x,y,z, max x,y,z                          */
#define TREE_DBG_COUNTS 6      /* uint32[n_groups][2] n_pp, n_pc of the last tree_force            */
#define TREE_DBG_GRID 7        /* float[10]     bbox lo[3], hi[3], cube origin[3], (float)k with side = 2^k */
#define TREE_DBG_ROPEN2 8      /* float[n_cells] squared opening radius of the last tree_force     */
#define TREE_DBG_SORTED_POS 9  /* float[N][4]   x,y,z,m in slot order                              */
#define TREE_DBG_LEVEL_OFFSETS 10 /* int32[24]  first cell id of each level 0..22, then n_cells   */
#define TREE_DBG_TASK_TRACE 11 /* uint32[n_tasks][4] per task of the last force pass: start ns since the
                                  pass began, duration ns, SM id, group | part << 26 (scheduling trace) */
#define TREE_DBG_TIGHT 12      /* float[n_cells][7] TREE_MAC_BMAX only: tight box lo x,y,z, hi x,y,z, bounding radius b */
int tree_get_debug(tree_ctx *t, int what, void *dst, long long *count);

/* Timings of the last tree_build / tree_force / tree_leapfrog in milliseconds (CUDA events on the
 * context's stream) and interaction totals of the last force pass, to HOST memory.
 * ms[TREE_NPHASE]: see TREE_PH_*.  n_pp / n_pc = sum over groups of group size x list length
 * ("as recorded during execution").  Synchronises. */
#define TREE_PH_KEYS 0     /* bbox + grid + keys (tree_leapfrog: grid + keys; its bbox is fused into the kick/drift pass) */
#define TREE_PH_SORT 1     /* radix sort of (key, index)         */
#define TREE_PH_PERMUTE 2  /* gather the particles (tree_leapfrog: positions, velocities, caller indices) into slot order */
#define TREE_PH_BUILD 3    /* octree construction + linking      */
#define TREE_PH_MOMENTS 4  /* groups + multipole moments         */
#define TREE_PH_OPENING 5  /* opening radii for theta            */
#define TREE_PH_WALK 6     /* the fused walk + force kernel only */
#define TREE_PH_UNPERMUTE 7 /* results to the caller's arrays as a pass of its own (sharded passes; tree_force on one context writes them in the walk's epilogue: 0) */
#define TREE_PH_INTEGRATE 8 /* leapfrog: kick + drift + bbox pass (the closing kick runs in the walk's epilogue; sharded
                               passes kick in a pass of their own after the barrier) */
#define TREE_PH_SCHED 9    /* counting walk + task list (cost-aware scheduling of the force walk) */
#define TREE_PH_TOTAL 10   /* sum of the above for the last call sequence */
#define TREE_NPHASE 11
int tree_get_stats(tree_ctx *t, double *ms, unsigned long long *n_pp, unsigned long long *n_pc);

/* ---- sharded force pass over several GPUs of one NVLink / NVSwitch node ------------------------
 * PAPER.md section III-B (L81-125) cuts the Peano-Hilbert curve into one piece per GPU (L93-97),
 * balances the pieces by the flops of the tree-walk (L107) and exchanges pruned trees over MPI
 * (L111-119) because node memory and network were the limits of 2014.  Here every
 * context of a node holds ALL N particles and builds the same tree (the build is ~3 % of a step on
 * this hardware); what is cut is the force pass: `world` contexts (one per GPU, one process each, or
 * several in one process) share one pass, context `rank` walking one contiguous range of groups of
 * the PH-sorted order with ~1/world of the estimated walk cost, and the walk kernel stores each
 * group's accelerations, potentials and interaction counts straight into the result buffers of
 * every attached context over NVLink (peer stores): there is no separate collective.  The one
 * exchange step of a force pass is a barrier between its two halves, which the CALLER provides
 * (e.g. one NCCL all-reduce on the contexts' streams; the binding's ShardedTree does that):
 *     tree_force_begin on every context  ->  barrier  ->  tree_force_end on every context.
 * Results are those of the same pass on one context up to the order of a few partial sums (the task
 * list differs); interaction counts per group are identical.
 *
 * Set-up, once, in this order: tree_reserve (buffers for the largest N) -> tree_shard_config ->
 * tree_shard_export / exchange the blobs / tree_shard_attach for every other rank (or
 * tree_shard_attach_local for contexts of the same process).  With world > 1, tree_force and
 * tree_leapfrog return TREE_ERR_ORDER (they cannot contain the barrier) and a tree_build beyond the
 * reserved capacity returns TREE_ERR_ORDER (it would invalidate the exported buffers). */
#define TREE_SHARD_MAX_WORLD 16
#define TREE_SHARD_HANDLE_BYTES 128

/* Allocate the particle-sized buffers for up to N particles now (they are otherwise grown by
 * tree_build). */
int tree_reserve(tree_ctx *t, long long N);
/* This context is `rank` of `world` (1 <= world <= TREE_SHARD_MAX_WORLD); world = 1 undoes it.  Synchronises the
 * stream.  A pass writes into one of two result buffers chosen by the parity of the context's pass count, and peers
 * store into the same parity: every call of tree_shard_config therefore restarts that count (and forgets the last
 * force: tree_get_state(acc) / tree_leapfrog need a new force pass), so that contexts with different histories can
 * share a pass.  From then on all contexts of a world must run the same sequence of passes. */
int tree_shard_config(tree_ctx *t, int rank, int world);
/* Write this context's result-buffer handle (a CUDA IPC handle and the reserved sizes) to
 * HOST memory handle[TREE_SHARD_HANDLE_BYTES].  Needs tree_reserve. */
int tree_shard_export(tree_ctx *t, void *handle);
/* Map the result buffers of context `peer_rank` living in ANOTHER process from its exported
 * HOST blob (cudaIpcOpenMemHandle; the GPUs must be peer-capable).  The peer must have reserved
 * the same N with the same group size. */
int tree_shard_attach(tree_ctx *t, int peer_rank, const void *handle);
/* Same for a context of THIS process (any device; peer access is enabled if needed). */
int tree_shard_attach_local(tree_ctx *t, int peer_rank, tree_ctx *peer);
/* First half of tree_force: opening radii, cost estimate, partition, task list, fused walk+force
 * over this context's range, results stored into every attached context.  Asynchronous. */
int tree_force_begin(tree_ctx *t, float theta, float eps);
/* Second half, after the caller's barrier: results to caller order (acc, pot as in tree_force). */
int tree_force_end(tree_ctx *t, float *acc, float *pot);
/* tree_leapfrog of a sharded context, in three parts around TWO barriers of the caller:
 *     tree_leapfrog_begin  kick, drift, bounding box, keys of all N; then the sort is cut by KEY RANGE (PAPER.md L93-97:
 *                          contiguous pieces of the PH curve): the keys at the slot boundaries N r / world of the previous
 *                          sorted order are splitters every context holds, context r sorts only the particles whose new
 *                          key falls into its range and stores the sorted run at its offset into every context
 *     -> barrier
 *     tree_leapfrog_mid    gather into the new order, octree, moments, tree_force_begin
 *     -> barrier
 *     tree_leapfrog_end    tree_force_end, kick.
 * On a context that is not sharded (world = 1) tree_leapfrog_begin does the first two parts and tree_leapfrog_mid
 * returns at once. */
int tree_leapfrog_begin(tree_ctx *t, float dt);
int tree_leapfrog_mid(tree_ctx *t);
int tree_leapfrog_end(tree_ctx *t);
/* The range of groups [*g_lo, *g_hi) and of slots [*s_lo, *s_hi) this context walked in the last
 * pass, to HOST memory (any pointer may be NULL).  Synchronises. */
int tree_shard_range(tree_ctx *t, long long *g_lo, long long *g_hi, long long *s_lo, long long *s_hi);

/* Measurement aid: the FP32 FMA rate in TFLOP/s this GPU sustains on register operands
 * (a short register-only FFMA kernel, best of 3), written to a HOST double: the measured denominator
 * reported beside the nominal FP32 peak in the roofline of the fused walk+force kernel.  Synchronises. */
int tree_fp32_peak(tree_ctx *t, double *tflops);

/* Measurement aid: the walk and the evaluation of the LAST force pass again, as two
 * kernels with the interaction lists going through global memory (one warp per group, groups in descending cost, no
 * splitting; needs an unsharded context, group size 64 and lists below 2^32 entries: N <= ~50 M).  ms[0] = the walk
 * alone (HOST double[2]), ms[1] = the evaluation alone, best of 3; *max_rel = largest relative deviation of its
 * accelerations from the fused pass's (HOST).  The evaluation alone bounds what separating walker and evaluator warps
 * could reach.  Allocates and frees its own buffers; synchronises. */
int tree_measure_listeval(tree_ctx *t, double *ms, double *max_rel);

/* ---- an entry point that allocates nothing -----------------------------------------------------
 * For callers that cannot call cudaMalloc (code under CUDA stream capture, tight serving loops, harnesses that forbid
 * it): the energy sums of tree_energy -- kinetic = sum 1/2 m v^2, potential = 1/2 sum m phi (the diagnostics of a
 * leapfrog run), FP64 sums of FP32 inputs -- without a context and without any allocation.  The scratch
 * tree_energy keeps in the context's cudaMalloc'ed buffers is here a fixed device array inside the library image
 * (512.25 KiB; every GPU that loads libbhtree.so holds it until the process exits), hence the limit
 *     N <= TREE_ENERGY_STATIC_MAX_N = 134,217,728 (32,768 partial sums of 4,096 particles each);
 * a larger N returns TREE_ERR_ARG with a text that says so (use tree_energy there).
 *   device       CUDA device the pointers live on (0..63); the caller's current device is restored
 *   cuda_stream  a cudaStream_t (may be NULL); the call enqueues one 4-byte cudaMemsetAsync and one kernel on it and
 *                returns without waiting; it calls no cudaMalloc, cudaFree or allocating library routine
 *   mass         DEV float[N]
 *   vel          DEV float[N][3] or NULL (kinetic = 0)
 *   pot          DEV float[N] or NULL (potential = 0): phi_i as tree_force / tree_get_state return it, same order as mass
 *   out          DEV double[2]: out[0] = kinetic, out[1] = potential, overwritten when the kernel has run
 *   N = 0        set-up only (asks the driver once per device for the scratch address; every pointer may be NULL):
 *                call it once before a stream capture begins, since the first call on a device may load the module
 * The sums are added in a fixed order: the same inputs give the same bits on every call, and agree with tree_energy
 * (atomic FP64 adds in arrival order) to rounding, ~1e-15 relative.
 * All calls on a device share the one scratch array, which keeps the last call's contents; the call clears the word
 * that must start at zero.  Calls that OVERLAP on the GPU (different streams, or two host threads on one device) race on
 * it and give wrong sums: order them on one stream or with events.
 * Errors: TREE_ERR_ARG / TREE_ERR_CUDA; text via tree_energy_static_error() (per host thread, "" after a success). */
#define TREE_ENERGY_STATIC_MAX_N 134217728LL
int tree_energy_static(int device, void *cuda_stream, const float *mass, const float *vel, const float *pot,
                       long long N, double *out);
const char *tree_energy_static_error(void);

/* Number of kernels this library launched on the context since tree_create (for accounting). */
long long tree_launch_count(const tree_ctx *t);

/* Text of the last error on this context ("" if none). Never NULL for a non-NULL context. */
const char *tree_last_error(const tree_ctx *t);

#ifdef __cplusplus
}
#endif
#endif /* BHTREE_TREE_H */
