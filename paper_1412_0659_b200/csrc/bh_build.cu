// Tree-build kernels (sm_100a): bounding box, Peano-Hilbert keys, radix sort, permutation,
// octree construction, groups, multipole moments.  HBM-bandwidth-bound phases.
// Compiled with -fmad=false: every FP operation that feeds an integer decision or a stored moment
// is a single IEEE operation in a fixed order (S9, S13).
#include "bh_common.cuh"

#define BH_TRY_RC(x) do { int _rc = (x); if (_rc) return _rc; } while (0)

namespace bh {

// ------------------------------------------------------------------------------------------
// small device helpers
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ int enc_f(float f) {  // order-preserving float -> int
  int i = __float_as_int(f);
  return i >= 0 ? i : i ^ 0x7fffffff;
}
__device__ __forceinline__ float dec_f(int i) { return __int_as_float(i >= 0 ? i : i ^ 0x7fffffff); }

__device__ __forceinline__ unsigned warp_incl_scan(unsigned v, int lane) {
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    unsigned n = __shfl_up_sync(0xffffffffu, v, o);
    if (lane >= o) v += n;
  }
  return v;
}

// Grid index of one coordinate (reading S9): one FP32 subtraction, exact power-of-two
// scale, floor, clamp to [0, 2^21).
__device__ __forceinline__ int grid_coord(float x, float o, float inv) {
  float t = __fsub_rn(x, o);
  float u = __fmul_rn(t, inv);
  float f = floorf(u);
  return (f < 0.0f) ? 0 : (f >= 2097152.0f ? 2097151 : (int)f);
}

// ------------------------------------------------------------------------------------------
// a1: bounding box (+ packing the caller's arrays into float4 x,y,z,m)
// ------------------------------------------------------------------------------------------
__global__ void info_reset_kernel(DevInfo *info) {
  if (threadIdx.x == 0) {
    for (int d = 0; d < 3; ++d) { info->lo_enc[d] = 0x7fffffff; info->hi_enc[d] = (int)0x80000000; }
    info->nonfinite = 0;
  }
}

// block-wide min/max of a per-thread box and OR of the non-finite flags, merged into info by integer atomics
__device__ __forceinline__ void block_bbox_reduce(float (&lo)[3], float (&hi)[3], int bad, DevInfo *info) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      lo[d] = fminf(lo[d], __shfl_xor_sync(0xffffffffu, lo[d], o));
      hi[d] = fmaxf(hi[d], __shfl_xor_sync(0xffffffffu, hi[d], o));
    }
    bad |= __shfl_xor_sync(0xffffffffu, bad, o);
  }
  __shared__ float s_lo[8][3], s_hi[8][3];
  __shared__ int s_bad[8];
  int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (lane == 0) {
    for (int d = 0; d < 3; ++d) { s_lo[w][d] = lo[d]; s_hi[w][d] = hi[d]; }
    s_bad[w] = bad;
  }
  __syncthreads();
  if (threadIdx.x < 3) {
    int d = threadIdx.x;
    float l = s_lo[0][d], h = s_hi[0][d];
    for (int k = 1; k < 8; ++k) { l = fminf(l, s_lo[k][d]); h = fmaxf(h, s_hi[k][d]); }
    atomicMin(&info->lo_enc[d], enc_f(l));
    atomicMax(&info->hi_enc[d], enc_f(h));
  }
  if (threadIdx.x == 3) {
    int b = 0;
    for (int k = 0; k < 8; ++k) b |= s_bad[k];
    if (b) atomicOr(&info->nonfinite, 1);
  }
}

template <bool PACK>
__global__ void __launch_bounds__(256) bbox_kernel(const float *__restrict__ pos, const float *__restrict__ mass,
                                                   float4 *__restrict__ posm, long long N, DevInfo *info) {
  float lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY};
  int bad = 0;
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x) {
    float4 p;
    if (PACK) {
      p.x = pos[3 * i]; p.y = pos[3 * i + 1]; p.z = pos[3 * i + 2]; p.w = mass[i];
      posm[i] = p;
    } else {
      p = posm[i];
    }
    bad |= !(isfinite(p.x) && isfinite(p.y) && isfinite(p.z) && isfinite(p.w));
    lo[0] = fminf(lo[0], p.x); hi[0] = fmaxf(hi[0], p.x);
    lo[1] = fminf(lo[1], p.y); hi[1] = fmaxf(hi[1], p.y);
    lo[2] = fminf(lo[2], p.z); hi[2] = fmaxf(hi[2], p.z);
  }
  block_bbox_reduce(lo, hi, bad, info);
}

// a12 + a1 fused (tree_leapfrog): v = fma(a, dt/2, v); x = fma(v, dt, x) on the slot-order state, and the bounding box of
// the new positions in the same pass (48 B read, 32 B written per particle; T12, "step pipeline").
__global__ void __launch_bounds__(256) kick_drift_bbox_kernel(float4 *__restrict__ spos, float4 *__restrict__ svel,
                                                              const float4 *__restrict__ sacc, long long N, float hdt,
                                                              float dt, DevInfo *info) {
  float lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY};
  int bad = 0;
  const bool frozen = info->cells_overflow != 0;  // a failed asynchronous rebuild freezes the state (tree.h): bbox only
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x) {
    float4 p = spos[i];
    if (!frozen) {
      float4 v = svel[i];
      const float4 a = sacc[i];
      v.x = __fmaf_rn(a.x, hdt, v.x); v.y = __fmaf_rn(a.y, hdt, v.y); v.z = __fmaf_rn(a.z, hdt, v.z);
      p.x = __fmaf_rn(v.x, dt, p.x); p.y = __fmaf_rn(v.y, dt, p.y); p.z = __fmaf_rn(v.z, dt, p.z);
      svel[i] = v;
      spos[i] = p;
    }
    bad |= !(isfinite(p.x) && isfinite(p.y) && isfinite(p.z) && isfinite(p.w));
    lo[0] = fminf(lo[0], p.x); hi[0] = fmaxf(hi[0], p.x);
    lo[1] = fminf(lo[1], p.y); hi[1] = fmaxf(hi[1], p.y);
    lo[2] = fminf(lo[2], p.z); hi[2] = fmaxf(hi[2], p.z);
  }
  block_bbox_reduce(lo, hi, bad, info);
}

// a2 (first half): cube centred on the bbox, side = smallest power of two > extent (S9).
__global__ void grid_kernel(DevInfo *info) {
  if (threadIdx.x != 0) return;
  double ext = 0.0;
  float lo[3], hi[3];
  for (int d = 0; d < 3; ++d) {
    lo[d] = dec_f(info->lo_enc[d]); hi[d] = dec_f(info->hi_enc[d]);
    info->lo[d] = lo[d]; info->hi[d] = hi[d];
    double e = (double)hi[d] - (double)lo[d];
    if (e > ext) ext = e;
  }
  int k = 0;
  if (ext > 0.0) { int e; frexp(ext, &e); k = e; }
  if (!(ext >= 0.0) || !isfinite(ext)) { info->nonfinite = 1; k = 0; }
  if (info->nonfinite) info->nonfinite_sticky = 1;  // an asynchronous rebuild reports it at the next synchronising call
  info->k = k;
  double S = ldexp(1.0, k);
  for (int d = 0; d < 3; ++d) {
    double c = 0.5 * ((double)lo[d] + (double)hi[d]);
    info->origin[d] = (float)(c - 0.5 * S);
  }
  info->inv = ldexpf(1.0f, KEY_BITS - k);
}

// a2: Peano-Hilbert key by a 24-state x 8-octant table generated on the host from the
// Gray-code/rotation recurrence (T3). Table entry = digit | next_state << 3.
// The kernel walks THREE levels per table step: a 24 x 512 table (three digits | next_state << 9; built once on the
// host from the 8-octant table, build_hilbert_lut3; every block copies its 24 KB into shared memory) indexed by state
// and by 3 bits of each grid coordinate, z | y | x, so the coordinates are never interleaved: a key costs 7 dependent
// shared-memory look-ups of ~12 instructions each (round 2 (a): 10 + 1 look-ups over Morton-interleaved coordinates,
// 205 instructions per key, of which the interleaving took 120; the kernel is bound by instruction issue, not by HBM).
__global__ void __launch_bounds__(256) keys_kernel(const float4 *__restrict__ posm, long long N,
                                                   const DevInfo *__restrict__ info, const uint16_t *__restrict__ lut3_g,
                                                   uint64_t *__restrict__ key, uint32_t *__restrict__ idx) {
  __shared__ __align__(16) uint16_t lut3[HLUT3_ENTRIES];
  for (int e = threadIdx.x; e < HLUT3_ENTRIES / 8; e += blockDim.x)
    reinterpret_cast<uint4 *>(lut3)[e] = reinterpret_cast<const uint4 *>(lut3_g)[e];
  __syncthreads();
  const float ox = info->origin[0], oy = info->origin[1], oz = info->origin[2], inv = info->inv;
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x) {
    float4 p = posm[i];
    const unsigned ix = grid_coord(p.x, ox, inv), iy = grid_coord(p.y, oy, inv) << 3, iz = grid_coord(p.z, oz, inv) << 6;
    unsigned st = 0, h[3] = {0u, 0u, 0u};  // 27 + 27 + 9 bits of the key
#pragma unroll
    for (int step = 0; step < 7; ++step) {  // levels (b+2, b+1, b), b = 18, 15, .., 0
      const int b = 18 - 3 * step;
      const unsigned t = ((ix >> b) & 7u) | ((iy >> b) & 0x38u) | ((iz >> b) & 0x1c0u);
      const unsigned v = lut3[st * 512 + t];
      h[step / 3] = (h[step / 3] << 9) | (v & 511u);
      st = v >> 9;
    }
    key[i] = ((uint64_t)h[0] << 36) | ((uint64_t)h[1] << 9) | (uint64_t)h[2];
    if (idx) idx[i] = (uint32_t)i;
  }
}

// ------------------------------------------------------------------------------------------
// device-wide exclusive scan of uint32 (in place): reduce -> scan block sums -> apply
// ------------------------------------------------------------------------------------------
constexpr int SCAN_THREADS = 512;
constexpr int SCAN_IPT = 8;
constexpr int SCAN_TILE = SCAN_THREADS * SCAN_IPT;

__device__ __forceinline__ unsigned block_excl_scan(unsigned v, unsigned *total, unsigned *s_w) {
  // exclusive scan of one value per thread over the block (SCAN_THREADS threads)
  int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  unsigned inc = warp_incl_scan(v, lane);
  if (lane == 31) s_w[w] = inc;
  __syncthreads();
  if (w == 0) {
    unsigned x = (lane < SCAN_THREADS / 32) ? s_w[lane] : 0;
    unsigned xi = warp_incl_scan(x, lane);
    s_w[lane] = xi - x;
    if (lane == 31) s_w[32] = xi;
  }
  __syncthreads();
  unsigned r = inc - v + s_w[w];
  if (total) *total = s_w[32];
  return r;
}

__global__ void __launch_bounds__(SCAN_THREADS) scan_reduce_kernel(const uint32_t *__restrict__ a, long long n,
                                                                    uint32_t *__restrict__ blk) {
  __shared__ unsigned s_w[33];
  long long base = (long long)blockIdx.x * SCAN_TILE + threadIdx.x * SCAN_IPT;
  unsigned s = 0;
#pragma unroll
  for (int k = 0; k < SCAN_IPT; ++k) if (base + k < n) s += a[base + k];
  unsigned tot;
  block_excl_scan(s, &tot, s_w);
  if (threadIdx.x == 0) blk[blockIdx.x] = tot;
}

__global__ void __launch_bounds__(SCAN_THREADS) scan_blocks_kernel(uint32_t *__restrict__ blk, int nblk,
                                                                    uint32_t *__restrict__ total_out) {
  __shared__ unsigned s_w[33];
  unsigned carry = 0;
  for (int b0 = 0; b0 < nblk; b0 += SCAN_THREADS) {
    int i = b0 + threadIdx.x;
    unsigned v = (i < nblk) ? blk[i] : 0;
    unsigned tot;
    unsigned e = block_excl_scan(v, &tot, s_w);
    if (i < nblk) blk[i] = e + carry;
    carry += tot;
    __syncthreads();
  }
  if (threadIdx.x == 0 && total_out) *total_out = carry;
}

__global__ void __launch_bounds__(SCAN_THREADS) scan_apply_kernel(uint32_t *__restrict__ a, long long n,
                                                                   const uint32_t *__restrict__ blk) {
  __shared__ unsigned s_w[33];
  long long base = (long long)blockIdx.x * SCAN_TILE + threadIdx.x * SCAN_IPT;
  unsigned v[SCAN_IPT], s = 0;
#pragma unroll
  for (int k = 0; k < SCAN_IPT; ++k) { v[k] = (base + k < n) ? a[base + k] : 0; s += v[k]; }
  unsigned e = block_excl_scan(s, nullptr, s_w) + blk[blockIdx.x];
#pragma unroll
  for (int k = 0; k < SCAN_IPT; ++k) {
    if (base + k < n) a[base + k] = e;
    e += v[k];
  }
}

int device_excl_scan(tree_ctx *t, uint32_t *a, long long n, uint32_t *total_out) {
  int nblk = (int)((n + SCAN_TILE - 1) / SCAN_TILE);
  scan_reduce_kernel<<<nblk, SCAN_THREADS, 0, t->stream>>>(a, n, t->b.scan_blk);
  BH_LAUNCH_CHECK("scan_reduce");
  scan_blocks_kernel<<<1, SCAN_THREADS, 0, t->stream>>>(t->b.scan_blk, nblk, total_out);
  BH_LAUNCH_CHECK("scan_blocks");
  scan_apply_kernel<<<nblk, SCAN_THREADS, 0, t->stream>>>(a, n, t->b.scan_blk);
  BH_LAUNCH_CHECK("scan_apply");
  return 0;
}

// ------------------------------------------------------------------------------------------
// a3: stable LSD radix sort of (key 64-bit, index 32-bit), 8 bits per pass, 8 passes.
// ------------------------------------------------------------------------------------------
constexpr int RADIX = 256;

// ------------------------------------------------------------------------------------------
// One-sweep form: one pass over the keys builds the 8 digit histograms; each of the 8 passes
// is then ONE kernel that ranks a tile, obtains the tile's global digit offsets by decoupled
// look-back over the preceding tiles' status words, and scatters. Per pass 12 B read + 12 B
// written per particle (+ 2 KB of status per 2048-key tile); 10 launches instead of 40.
// Tiles take their index from an atomic ticket, so a tile only ever waits for tiles that are
// already running or finished. Status word: flag (2 bits) | epoch (30 bits) | value (32 bits);
// the epoch changes every pass, so the array is never cleared.
// ------------------------------------------------------------------------------------------
constexpr int OS_THREADS = 256;
constexpr int OS_IPT = 8;
constexpr int OS_TILE = OS_THREADS * OS_IPT;  // 2048
constexpr int OS_WARPS = OS_THREADS / 32;
constexpr int OS_MINB = 5;  // resident blocks per SM (shared memory allows 6)
constexpr unsigned long long OS_LOCAL = 1ull << 62, OS_INCL = 2ull << 62;
constexpr int OS_LOOK = 8;  // status words one thread keeps in flight during the look-back (4 / 8 / 16 / 32 measured: 11.39 /
                            // 11.30 / 11.66 / 27.1 ms per sort at N = 134 M; 32 spills)

// n_dev != nullptr: the number of keys is *n_dev (a bucket of a sharded step, known only on the device)
__global__ void __launch_bounds__(256) sort_hist8_kernel(const uint64_t *__restrict__ key, long long N,
                                                         const unsigned *__restrict__ n_dev,
                                                         uint32_t *__restrict__ ghist /*[8][256]*/) {
  __shared__ unsigned h[8 * RADIX];
  if (n_dev) N = *n_dev;
  for (int i = threadIdx.x; i < 8 * RADIX; i += blockDim.x) h[i] = 0;
  __syncthreads();
  for (long long p = blockIdx.x * (long long)blockDim.x + threadIdx.x; p < N; p += (long long)gridDim.x * blockDim.x) {
    const uint64_t k = key[p];
#pragma unroll
    for (int d = 0; d < 8; ++d) atomicAdd(&h[d * RADIX + ((unsigned)(k >> (8 * d)) & 255u)], 1u);
  }
  __syncthreads();
  for (int i = threadIdx.x; i < 8 * RADIX; i += blockDim.x) {
    const unsigned v = h[i];
    if (v) atomicAdd(&ghist[i], v);
  }
}

// exclusive scan of each of the 8 histograms (block p handles pass p); also clears the tile tickets
__global__ void __launch_bounds__(RADIX) sort_scan8_kernel(uint32_t *__restrict__ ghist, uint32_t *__restrict__ ticket) {
  __shared__ unsigned s_w[9];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const unsigned v = ghist[blockIdx.x * RADIX + threadIdx.x];
  const unsigned inc = warp_incl_scan(v, lane);
  if (lane == 31) s_w[w] = inc;
  __syncthreads();
  if (threadIdx.x == 0) {
    unsigned run = 0;
    for (int k = 0; k < RADIX / 32; ++k) { unsigned c = s_w[k]; s_w[k] = run; run += c; }
    ticket[blockIdx.x] = 0;
  }
  __syncthreads();
  ghist[blockIdx.x * RADIX + threadIdx.x] = inc - v + s_w[w];
}

__device__ __forceinline__ unsigned long long ld_status(const unsigned long long *p) {
  unsigned long long v;
  asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_status(unsigned long long *p, unsigned long long v) {
  asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

struct OsSmem {
  uint64_t key[OS_TILE];
  uint32_t val[OS_TILE];
  unsigned wc[OS_WARPS][RADIX];
  unsigned dstart[RADIX];
  unsigned gbase[RADIX];
  unsigned tile;
};

__global__ void __launch_bounds__(OS_THREADS, OS_MINB) sort_onesweep_kernel(const uint64_t *__restrict__ kin,
                                                                   const uint32_t *__restrict__ vin,
                                                                   uint64_t *__restrict__ kout, uint32_t *__restrict__ vout,
                                                                   const uint32_t *__restrict__ gscan /*[256] of this pass*/,
                                                                   uint32_t *__restrict__ ticket,
                                                                   unsigned long long *__restrict__ status /*[tiles][256]*/,
                                                                   unsigned long long epoch, int shift, long long N,
                                                                   const unsigned *__restrict__ n_dev) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  OsSmem &sm = *reinterpret_cast<OsSmem *>(smem_raw);
  const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const unsigned lt = (1u << lane) - 1u;
  if (n_dev) N = *n_dev;  // the grid covers an upper bound; tiles past the end take a ticket and leave
  if (threadIdx.x == 0) sm.tile = atomicAdd(ticket, 1u);
  for (int i = lane; i < RADIX; i += 32) sm.wc[w][i] = 0;
  __syncthreads();
  const unsigned tile = sm.tile;
  const long long base = (long long)tile * OS_TILE;
  if (base >= N) return;  // block-uniform; nobody looks back at a tile that does not exist
  uint64_t key[OS_IPT];
  unsigned rank[OS_IPT];
  // warp-striped: warp w owns items [w*256, w*256+256) of the tile, item k of lane l at k*32+l
#pragma unroll
  for (int k = 0; k < OS_IPT; ++k) {
    const long long p = base + w * (32 * OS_IPT) + k * 32 + lane;
    const bool valid = p < N;
    key[k] = valid ? kin[p] : 0;
  }
#pragma unroll
  for (int k = 0; k < OS_IPT; ++k) {
    const long long p = base + w * (32 * OS_IPT) + k * 32 + lane;
    const bool valid = p < N;
    const unsigned d = (unsigned)(key[k] >> shift) & 255u;
    const unsigned act = __ballot_sync(0xffffffffu, valid);
    // lanes with the same digit: one ballot per digit bit (MATCH.ANY takes one round per distinct value in the warp: with
    // 8-bit digits of well-mixed keys that is ~28 rounds, and the warps queued behind it)
    unsigned peers = act, c0 = 0;
#pragma unroll
    for (int b = 0; b < 8; ++b) {
      const bool bit = (d >> b) & 1u;
      const unsigned v = __ballot_sync(0xffffffffu, bit);
      peers &= bit ? v : ~v;
    }
    if (valid) c0 = sm.wc[w][d];
    __syncwarp();
    if (valid && lane == 31 - __clz(peers)) sm.wc[w][d] = c0 + __popc(peers);
    __syncwarp();
    rank[k] = c0 + __popc(peers & lt);
  }
  __syncthreads();
  // thread d: digit d's exclusive prefix over the warps and the tile's count, published at once (LOCAL) so that later
  // tiles can look past this one while it is still busy
  unsigned my_count = 0;
  {
    const unsigned d = threadIdx.x;
    unsigned run = 0;
#pragma unroll
    for (int ww = 0; ww < OS_WARPS; ++ww) {
      const unsigned c = sm.wc[ww][d];
      sm.wc[ww][d] = run;
      run += c;
    }
    sm.dstart[d] = run;  // tile count of digit d (scanned below)
    my_count = run;
    if (tile > 0) st_status(status + (size_t)tile * RADIX + d, OS_LOCAL | (epoch << 32) | run);
  }
  __syncthreads();
  if (w == 0) {  // exclusive scan of the 256 tile counts
    unsigned v[8], s = 0;
#pragma unroll
    for (int j = 0; j < 8; ++j) { v[j] = sm.dstart[lane * 8 + j]; s += v[j]; }
    unsigned e = warp_incl_scan(s, lane) - s;
#pragma unroll
    for (int j = 0; j < 8; ++j) { sm.dstart[lane * 8 + j] = e; e += v[j]; }
  }
  __syncthreads();
  // keys and payloads to their place in the tile's digit order (shared memory) BEFORE the look-back: the key and rank
  // registers are dead afterwards, so the look-back can keep OS_LOOK status words in flight without spilling
#pragma unroll
  for (int k = 0; k < OS_IPT; ++k) {
    const long long p = base + w * (32 * OS_IPT) + k * 32 + lane;
    if (p < N) {
      const unsigned d = (unsigned)(key[k] >> shift) & 255u;
      const unsigned q = sm.dstart[d] + sm.wc[w][d] + rank[k];
      sm.key[q] = key[k];
      sm.val[q] = vin ? vin[p] : (uint32_t)p;  // payload read late: 8 registers fewer while ranking
    }
  }
  // thread d: look back over the preceding tiles, OS_LOOK status words in flight at a time
  {
    const unsigned d = threadIdx.x;
    unsigned long long *mine = status + (size_t)tile * RADIX + d;
    const unsigned long long tag = epoch << 32;
    const unsigned tag_hi = (unsigned)epoch;  // epoch < 2^30: the high word of a status word of this pass is flag << 30 | epoch
    unsigned excl = 0;
    if (tile > 0) {
      bool done = false;
      for (long long q = (long long)tile - 1; q >= 0 && !done; q -= OS_LOOK) {
        unsigned long long v[OS_LOOK];
#pragma unroll
        for (int j = 0; j < OS_LOOK; ++j)
          v[j] = (q - j >= 0) ? ld_status(status + (size_t)(q - j) * RADIX + d) : (OS_INCL | tag);
        // the usual case: all OS_LOOK words were published long ago (a tile walks back over ~40 predecessors): sum the
        // local counts up to the first inclusive prefix without a branch per word
        bool all_ok = true;
#pragma unroll
        for (int j = 0; j < OS_LOOK; ++j) {
          const unsigned hi = (unsigned)(v[j] >> 32);
          all_ok = all_ok && (hi & 0x3fffffffu) == tag_hi && (hi >> 30) != 0u;
        }
        if (all_ok) {
#pragma unroll
          for (int j = 0; j < OS_LOOK; ++j) {
            excl += done ? 0u : (unsigned)v[j];
            done = done || (unsigned)(v[j] >> 62) == 2u;
          }
          continue;
        }
#pragma unroll
        for (int j = 0; j < OS_LOOK; ++j) {
          if (done) break;
          unsigned long long x = v[j];
          while ((x & 0x3fffffff00000000ull) != tag || (x >> 62) == 0ull) x = ld_status(status + (size_t)(q - j) * RADIX + d);
          excl += (unsigned)x;
          done = (x >> 62) == 2ull;
        }
      }
    }
    st_status(mine, OS_INCL | tag | (unsigned long long)(excl + my_count));
    sm.gbase[d] = gscan[d] + excl;
  }
  __syncthreads();
  const long long rem = N - base;
  const int cnt = rem < OS_TILE ? (int)rem : OS_TILE;
  for (int j = threadIdx.x; j < cnt; j += OS_THREADS) {
    const uint64_t kk = sm.key[j];
    const unsigned d = (unsigned)(kk >> shift) & 255u;
    const long long dst = (long long)sm.gbase[d] + (j - (int)sm.dstart[d]);
    kout[dst] = kk;
    vout[dst] = sm.val[j];
  }
}

// a4: gather the particles into slot order.
// tree_build: the sort's payload is the caller index (a stable sort of the caller-ordered keys: ties by caller index, S10).
__global__ void __launch_bounds__(256) permute_build_kernel(const float4 *__restrict__ posm, const uint32_t *__restrict__ sidx,
                                                            float4 *__restrict__ spos, uint32_t *__restrict__ order, long long N) {
  long long s = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (s < N) {
    const uint32_t i = sidx[s];
    spos[s] = posm[i];
    order[s] = i;
  }
}

// tree_leapfrog: the state lives in the slot order of the previous step and the sort's payload is the PREVIOUS SLOT, so the
// gathers below are nearly sequential (few particles change their place on the curve in one step).  The stable sort left
// equal keys (particles in one finest grid cell) in previous-slot order; S10 wants them by caller index, so a slot inside
// a run of equal keys ranks itself within the run by caller index (runs are short: pairs in the densest cells; the
// ranking is quadratic in the run length).
__global__ void __launch_bounds__(256) permute_step_kernel(const uint64_t *__restrict__ skey, const uint32_t *__restrict__ perm,
                                                           const float4 *__restrict__ pos_in, const float4 *__restrict__ vel_in,
                                                           const uint32_t *__restrict__ order_in, float4 *__restrict__ pos_out,
                                                           float4 *__restrict__ vel_out, uint32_t *__restrict__ order_out,
                                                           const float *__restrict__ amag_in, float *__restrict__ amag_out,
                                                           long long N) {
  const long long s = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (s >= N) return;
  const uint64_t k = skey[s];
  const uint32_t q = perm[s];
  const uint32_t me = order_in[q];
  long long dst = s;
  const bool tie_l = s > 0 && skey[s - 1] == k, tie_r = s + 1 < N && skey[s + 1] == k;
  if (tie_l || tie_r) {
    long long r0 = s, r1 = s + 1;
    while (r0 > 0 && skey[r0 - 1] == k) --r0;
    while (r1 < N && skey[r1] == k) ++r1;
    long long rank = 0;
    for (long long j = r0; j < r1; ++j) rank += order_in[perm[j]] < me;
    dst = r0 + rank;
  }
  pos_out[dst] = pos_in[q];
  vel_out[dst] = vel_in[q];
  order_out[dst] = me;
  if (amag_in) amag_out[dst] = amag_in[q];  // relative criterion: |a| of the last force pass travels with the particle
}

// ------------------------------------------------------------------------------------------
// a5: octree from the sorted keys, without a per-level pass over the particles.
// cd(p) = number of leading 3-bit digits shared by key[p-1] and key[p] (-1 at the ends).
// Slot s starts cells at levels L0(s) = cd(s)+1 .. Lleaf(s), where Lleaf(s) = 1 + (leaf_size-th
// largest "common digits with s" among the other particles), capped at 21: the level at which
// the cell around s first holds <= leaf_size particles (DESIGN.md §Tree construction).
// ------------------------------------------------------------------------------------------
constexpr int TREE_THREADS = 512;
constexpr int TREE_HALO = 32;  // >= max leaf_size

__device__ __forceinline__ int common_digits(const uint64_t *__restrict__ key, long long p, long long N) {
  if (p <= 0 || p >= N) return -1;
  uint64_t x = key[p - 1] ^ key[p];
  if (x == 0) return KEY_BITS;
  return (__clzll((long long)x) - 1) / 3;
}

__global__ void __launch_bounds__(TREE_THREADS) tree_levels_kernel(const uint64_t *__restrict__ skey, long long N,
                                                                    int leaf, int ntiles, uint16_t *__restrict__ lv,
                                                                    uint32_t *__restrict__ tilecnt) {
  __shared__ signed char cd[TREE_THREADS + 2 * TREE_HALO + 1];
  __shared__ unsigned cnt[NLEVELS];
  const long long base = (long long)blockIdx.x * TREE_THREADS;
  if (threadIdx.x < NLEVELS) cnt[threadIdx.x] = 0;
  for (int i = threadIdx.x; i < TREE_THREADS + 2 * TREE_HALO + 1; i += TREE_THREADS)
    cd[i] = (signed char)common_digits(skey, base - TREE_HALO + i, N);
  __syncthreads();
  long long s = base + threadIdx.x;
  if (s < N) {
    int i = threadIdx.x + TREE_HALO;
    int L0 = cd[i] + 1;
    int v = KEY_BITS;
    if (leaf == 16) {
      // the leaf-th largest of the two non-increasing sequences lm[j] = min(cd[i], .., cd[i-j+1]) and
      // rm[j] = min(cd[i+1], .., cd[i+j]) is max over k of min(lm[k], rm[leaf-k]) (lm[0] = rm[0] = KEY_BITS):
      // the value the merge walk below ends on, without its data-dependent selects
      int rm[17];
      rm[0] = KEY_BITS;
#pragma unroll
      for (int j = 1; j <= 16; ++j) rm[j] = min(rm[j - 1], (int)cd[i + j]);
      v = rm[16];
      int lm = KEY_BITS;
#pragma unroll
      for (int k = 1; k <= 16; ++k) {
        lm = min(lm, (int)cd[i - k + 1]);
        v = max(v, min(lm, rm[16 - k]));
      }
    } else {
      int lmin = KEY_BITS, rmin = KEY_BITS, li = i, ri = i + 1;
      for (int it = 0; it < leaf; ++it) {
        int cl = min(lmin, (int)cd[li]), cr = min(rmin, (int)cd[ri]);
        if (cl >= cr) { v = cl; lmin = cl; --li; } else { v = cr; rmin = cr; ++ri; }
      }
    }
    int Ll = min(MAX_LEVEL, v + 1);
    lv[s] = (uint16_t)(L0 | (Ll << 5));
    for (int l = L0; l <= Ll; ++l) atomicAdd(&cnt[l], 1u);
  }
  __syncthreads();
  if (threadIdx.x < NLEVELS) tilecnt[(long long)threadIdx.x * ntiles + blockIdx.x] = cnt[threadIdx.x];
}

// levels 0..ltop together hold at most this many cells: one block computes their moments (moments_top_kernel)
constexpr int MOMENTS_TOP_CELLS = 128;

// Level offsets, cell count, the top levels one block handles, and the capacity check of an asynchronous rebuild:
// `cells_bound` cells are allocated / launched for; a tree that needs more sets the sticky cells_overflow and every
// later kernel of the step pipeline does nothing (the host reports it at its next synchronising call, tree.h).
__global__ void tree_offsets_kernel(const uint32_t *__restrict__ scanned, int ntiles, const uint32_t *__restrict__ total,
                                    long long cells_bound, DevInfo *info) {
  __shared__ int off[NLEVELS + 1];
  int l = threadIdx.x;
  if (l < NLEVELS) off[l] = (int)scanned[(long long)l * ntiles];
  if (l == NLEVELS) off[NLEVELS] = (int)*total;
  __syncthreads();
  if (l <= NLEVELS) info->level_off[l] = off[l];
  if (l == 0) {
    const unsigned nc = (unsigned)off[NLEVELS];
    info->n_cells = (int)nc;
    if ((long long)nc > cells_bound && !info->cells_overflow) info->cells_overflow = nc;
    int ltop = -1;
    while (ltop + 1 <= MAX_LEVEL && off[ltop + 2] <= MOMENTS_TOP_CELLS) ++ltop;
    info->ltop = ltop;
  }
}

__global__ void __launch_bounds__(TREE_THREADS) tree_emit_kernel(const uint16_t *__restrict__ lv, long long N,
                                                                  int ntiles, const uint32_t *__restrict__ scanned,
                                                                  uint8_t *__restrict__ c_level,
                                                                  uint32_t *__restrict__ c_first,
                                                                  uint32_t *__restrict__ c_count,
                                                                  uint32_t *__restrict__ c_fcall,
                                                                  const DevInfo *__restrict__ info) {
  constexpr int NW = TREE_THREADS / 32;
  if (info->cells_overflow) return;
  __shared__ uint16_t lvs[TREE_THREADS + TREE_HALO + 1];
  __shared__ unsigned wbase[NLEVELS][NW];
  __shared__ unsigned wleaf[NW + 1];  // per warp: which of its slots start a leaf; [NW]: the same for the halo
  const long long base = (long long)blockIdx.x * TREE_THREADS;
  const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const unsigned lt = (1u << lane) - 1u;
  for (int i = threadIdx.x; i < TREE_THREADS + TREE_HALO + 1; i += TREE_THREADS) {
    long long p = base + i;
    lvs[i] = (p < N) ? lv[p] : (uint16_t)0;  // L0 = 0 terminates every rightward scan
  }
  __syncthreads();
  const long long s = base + threadIdx.x;
  const bool valid = s < N;
  const int me = lvs[threadIdx.x];
  const int L0 = valid ? (me & 31) : 99, Ll = valid ? (me >> 5) : -1;
  // levels at which any slot of this warp starts a cell: [lo, hi] (warp-uniform); the other levels count zero
  int lo = L0, hi = Ll;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    lo = min(lo, __shfl_xor_sync(0xffffffffu, lo, o));
    hi = max(hi, __shfl_xor_sync(0xffffffffu, hi, o));
  }
  if (lane < NLEVELS) wbase[lane][w] = 0;
  __syncwarp();
  for (int l = lo; l <= hi; ++l) {
    unsigned b = __ballot_sync(0xffffffffu, L0 <= l && l <= Ll);
    if (lane == 0) wbase[l][w] = __popc(b);
  }
  // a slot is the first of its leaf iff it starts a cell at all (L0 <= Ll): leaves tile the slots, so a leaf ends where
  // the next one starts.  One ballot per warp (and one for the halo); slots past N count as starts: they terminate.
  {
    const unsigned f = __ballot_sync(0xffffffffu, !valid || L0 <= Ll);
    if (lane == 0) wleaf[w] = f;
    if (w == 0) {
      const int h = lvs[TREE_THREADS + lane];
      const unsigned fh = __ballot_sync(0xffffffffu, (h & 31) <= (h >> 5));
      if (lane == 0) wleaf[NW] = fh;
    }
  }
  __syncthreads();
  if (threadIdx.x < NLEVELS) {
    unsigned run = scanned[(long long)threadIdx.x * ntiles + blockIdx.x];
    for (int ww = 0; ww < NW; ++ww) { unsigned c = wbase[threadIdx.x][ww]; wbase[threadIdx.x][ww] = run; run += c; }
  }
  __syncthreads();
  if (hi < 0) return;  // whole warp past the end (warp-uniform)
  if (lo > hi) return;
  unsigned bcur = __ballot_sync(0xffffffffu, L0 <= lo && lo <= Ll);
  for (int l = lo; l <= hi; ++l) {
    unsigned bnext = __ballot_sync(0xffffffffu, L0 <= l + 1 && l + 1 <= Ll);
    if (L0 <= l && l <= Ll) {
      unsigned id = wbase[l][w] + __popc(bcur & lt);
      unsigned child = wbase[l + 1][w] + __popc(bnext & lt);  // level 22 is empty: = n_cells
      unsigned cnt = 0;
      if (l == Ll) {  // leaf: extent = up to the next slot that starts a leaf (or N)
        const unsigned above = lane < 31 ? wleaf[w] >> (lane + 1) : 0u;
        const unsigned next = wleaf[w + 1];
        if (above) cnt = (unsigned)__ffs(above);
        else if (next) cnt = (unsigned)(31 - lane + __ffs(next));
        else {  // more than 32 slots: only a leaf of the deepest level can be that full (coincident keys)
          long long e = s + (32 - lane) + 32;
          while (e < N) {
            const int m = lv[e];
            if ((m & 31) <= (m >> 5)) break;
            ++e;
          }
          cnt = (unsigned)(e - s);
        }
      }
      c_level[id] = (uint8_t)l;
      c_first[id] = (uint32_t)s;
      c_count[id] = cnt;
      c_fcall[id] = child;
    }
    bcur = bnext;
  }
}

// child links: n_child(c) = fcall[c+1] - fcall[c]; 0 = leaf.
__global__ void __launch_bounds__(256) tree_link_kernel(const DevInfo *__restrict__ info, const uint32_t *__restrict__ c_first,
                                                        const uint32_t *__restrict__ c_count,
                                                        const uint32_t *__restrict__ c_fcall, uint2 *__restrict__ c_link) {
  if (info->cells_overflow) return;
  const long long n_cells = info->n_cells;
  long long c = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (c >= n_cells) return;
  unsigned f = c_fcall[c];
  unsigned nx = (c + 1 < n_cells) ? c_fcall[c + 1] : (unsigned)n_cells;
  unsigned nch = nx - f;
  c_link[c] = nch ? make_uint2(f, nch | LEAF_FLAG) : make_uint2(c_first[c], c_count[c]);
}

// ------------------------------------------------------------------------------------------
// a6: groups = runs of `group` consecutive slots, tight AABB. One warp per group.
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) groups_kernel(const float4 *__restrict__ spos, long long N, int group,
                                                     long long n_groups, float *__restrict__ gbox) {
  long long g = (blockIdx.x * (long long)blockDim.x + threadIdx.x) >> 5;
  int lane = threadIdx.x & 31;
  if (g >= n_groups) return;
  float lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY};
  for (int j = lane; j < group; j += 32) {
    long long s = g * group + j;
    if (s < N) {
      float4 p = spos[s];
      lo[0] = fminf(lo[0], p.x); hi[0] = fmaxf(hi[0], p.x);
      lo[1] = fminf(lo[1], p.y); hi[1] = fmaxf(hi[1], p.y);
      lo[2] = fminf(lo[2], p.z); hi[2] = fmaxf(hi[2], p.z);
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1)
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      lo[d] = fminf(lo[d], __shfl_xor_sync(0xffffffffu, lo[d], o));
      hi[d] = fmaxf(hi[d], __shfl_xor_sync(0xffffffffu, hi[d], o));
    }
  if (lane == 0) {
    float *o = gbox + 6 * g;
    o[0] = lo[0]; o[1] = lo[1]; o[2] = lo[2]; o[3] = hi[0]; o[4] = hi[1]; o[5] = hi[2];
  }
}

// ------------------------------------------------------------------------------------------
// a7: multipole moments of one level (leaves from particles, internal cells from their children,
// which are one level deeper and already done).  FP64 accumulation in slot order, one rounding to
// FP32 per stored value (S13).  Q = sum m d d^T about the FP32-rounded centre of mass (S4).
// ------------------------------------------------------------------------------------------
// One cell. `leaves` selects which kind of cell this call handles: leaves depend on the particles only and
// are all done by one launch; internal cells follow level by level, deepest first.
__device__ __forceinline__ void moments_cell(int c, int level, bool leaves, const DevInfo *__restrict__ info,
                                             const float4 *__restrict__ spos, const uint2 *__restrict__ c_link,
                                             const uint32_t *__restrict__ c_first, uint32_t *__restrict__ c_count,
                                             float4 *__restrict__ c_cm, float4 *__restrict__ c_qa,
                                             float4 *__restrict__ c_qb, float4 *__restrict__ c_tlo = nullptr,
                                             float4 *__restrict__ c_thi = nullptr) {
  const uint2 lk = c_link[c];
  if (leaves != !(lk.y & LEAF_FLAG)) return;
  double M = 0, s0 = 0, s1 = 0, s2 = 0;
  double Q0 = 0, Q1 = 0, Q2 = 0, Q3 = 0, Q4 = 0, Q5 = 0;
  float cx, cy, cz;
  if (!(lk.y & LEAF_FLAG)) {
    const unsigned f = lk.x, n = lk.y;
#pragma unroll 4
    for (unsigned p = f; p < f + n; ++p) {
      float4 q = spos[p];
      double m = (double)q.w;
      M = __dadd_rn(M, m);
      s0 = __dadd_rn(s0, __dmul_rn(m, (double)q.x));
      s1 = __dadd_rn(s1, __dmul_rn(m, (double)q.y));
      s2 = __dadd_rn(s2, __dmul_rn(m, (double)q.z));
    }
    cx = (float)(s0 / M); cy = (float)(s1 / M); cz = (float)(s2 / M);
#pragma unroll 4
    for (unsigned p = f; p < f + n; ++p) {
      float4 q = spos[p];
      double m = (double)q.w;
      double dx = __dsub_rn((double)q.x, (double)cx), dy = __dsub_rn((double)q.y, (double)cy),
             dz = __dsub_rn((double)q.z, (double)cz);
      double mx = __dmul_rn(m, dx), my = __dmul_rn(m, dy), mz = __dmul_rn(m, dz);
      Q0 = __dadd_rn(Q0, __dmul_rn(mx, dx)); Q1 = __dadd_rn(Q1, __dmul_rn(my, dy)); Q2 = __dadd_rn(Q2, __dmul_rn(mz, dz));
      Q3 = __dadd_rn(Q3, __dmul_rn(mx, dy)); Q4 = __dadd_rn(Q4, __dmul_rn(mx, dz)); Q5 = __dadd_rn(Q5, __dmul_rn(my, dz));
    }
  } else {
    const unsigned f = lk.x, n = lk.y & ~LEAF_FLAG;
    unsigned cnt = 0;
    for (unsigned ch = f; ch < f + n; ++ch) {
      float4 a = c_cm[ch];
      double m = (double)a.w;
      M = __dadd_rn(M, m);
      s0 = __dadd_rn(s0, __dmul_rn(m, (double)a.x));
      s1 = __dadd_rn(s1, __dmul_rn(m, (double)a.y));
      s2 = __dadd_rn(s2, __dmul_rn(m, (double)a.z));
      cnt += c_count[ch];
    }
    c_count[c] = cnt;
    cx = (float)(s0 / M); cy = (float)(s1 / M); cz = (float)(s2 / M);
    for (unsigned ch = f; ch < f + n; ++ch) {
      float4 a = c_cm[ch], qa = c_qa[ch], qb = c_qb[ch];
      double m = (double)a.w;
      double dx = __dsub_rn((double)a.x, (double)cx), dy = __dsub_rn((double)a.y, (double)cy),
             dz = __dsub_rn((double)a.z, (double)cz);
      double mx = __dmul_rn(m, dx), my = __dmul_rn(m, dy), mz = __dmul_rn(m, dz);
      Q0 = __dadd_rn(Q0, __dadd_rn((double)qa.x, __dmul_rn(mx, dx)));
      Q1 = __dadd_rn(Q1, __dadd_rn((double)qa.y, __dmul_rn(my, dy)));
      Q2 = __dadd_rn(Q2, __dadd_rn((double)qa.z, __dmul_rn(mz, dz)));
      Q3 = __dadd_rn(Q3, __dadd_rn((double)qb.x, __dmul_rn(mx, dy)));
      Q4 = __dadd_rn(Q4, __dadd_rn((double)qb.y, __dmul_rn(mx, dz)));
      Q5 = __dadd_rn(Q5, __dadd_rn((double)qb.z, __dmul_rn(my, dz)));
    }
  }
  // geometric centre of the octant from the grid coordinates of the first particle (T6)
  const float4 pf = spos[c_first[c]];
  const float inv = info->inv;
  const double lc = ldexp(1.0, info->k - level);
  const int sh = KEY_BITS - level;
  double qx = (double)(grid_coord(pf.x, info->origin[0], inv) >> sh);
  double qy = (double)(grid_coord(pf.y, info->origin[1], inv) >> sh);
  double qz = (double)(grid_coord(pf.z, info->origin[2], inv) >> sh);
  double gx = __dadd_rn((double)info->origin[0], __dmul_rn(__dadd_rn(qx, 0.5), lc));
  double gy = __dadd_rn((double)info->origin[1], __dmul_rn(__dadd_rn(qy, 0.5), lc));
  double gz = __dadd_rn((double)info->origin[2], __dmul_rn(__dadd_rn(qz, 0.5), lc));
  double ex = __dsub_rn((double)cx, gx), ey = __dsub_rn((double)cy, gy), ez = __dsub_rn((double)cz, gz);
  double del = __dsqrt_rn(__dadd_rn(__dadd_rn(__dmul_rn(ex, ex), __dmul_rn(ey, ey)), __dmul_rn(ez, ez)));
  if (c_tlo) {  // TREE_MAC_BMAX: tight box of the cell's particles (min / max are exact) and the bounding radius about
                // the FP32 centre of mass: e_d = max(c_d - lo_d, hi_d - c_d); b = sqrt(fma(ez, ez, fma(ey, ey, ex ex)))
    float lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY};
    if (!(lk.y & LEAF_FLAG)) {
      for (unsigned p = lk.x; p < lk.x + lk.y; ++p) {
        const float4 q = spos[p];
        lo[0] = fminf(lo[0], q.x); hi[0] = fmaxf(hi[0], q.x);
        lo[1] = fminf(lo[1], q.y); hi[1] = fmaxf(hi[1], q.y);
        lo[2] = fminf(lo[2], q.z); hi[2] = fmaxf(hi[2], q.z);
      }
    } else {
      const unsigned f = lk.x, n = lk.y & ~LEAF_FLAG;
      for (unsigned ch = f; ch < f + n; ++ch) {
        const float4 a = c_tlo[ch], b = c_thi[ch];
        lo[0] = fminf(lo[0], a.x); hi[0] = fmaxf(hi[0], b.x);
        lo[1] = fminf(lo[1], a.y); hi[1] = fmaxf(hi[1], b.y);
        lo[2] = fminf(lo[2], a.z); hi[2] = fmaxf(hi[2], b.z);
      }
    }
    const float e0 = fmaxf(__fsub_rn(cx, lo[0]), __fsub_rn(hi[0], cx));
    const float e1 = fmaxf(__fsub_rn(cy, lo[1]), __fsub_rn(hi[1], cy));
    const float e2 = fmaxf(__fsub_rn(cz, lo[2]), __fsub_rn(hi[2], cz));
    const float b2 = __fmaf_rn(e2, e2, __fmaf_rn(e1, e1, __fmul_rn(e0, e0)));
    c_tlo[c] = make_float4(lo[0], lo[1], lo[2], __fsqrt_rn(b2));
    c_thi[c] = make_float4(hi[0], hi[1], hi[2], 0.0f);
  }
  float q0 = (float)Q0, q1 = (float)Q1, q2 = (float)Q2;
  c_cm[c] = make_float4(cx, cy, cz, (float)M);
  c_qa[c] = make_float4(q0, q1, q2, (float)del);
  c_qb[c] = make_float4((float)Q3, (float)Q4, (float)Q5, __fadd_rn(__fadd_rn(q0, q1), q2));
}

// all leaves, any level (the level of a cell comes from c_level); the cell count is read on the device
__global__ void __launch_bounds__(128) moments_leaf_kernel(const DevInfo *__restrict__ info,
                                                           const float4 *__restrict__ spos, const uint2 *__restrict__ c_link,
                                                           const uint8_t *__restrict__ c_level,
                                                           const uint32_t *__restrict__ c_first,
                                                           uint32_t *__restrict__ c_count, float4 *__restrict__ c_cm,
                                                           float4 *__restrict__ c_qa, float4 *__restrict__ c_qb,
                                                           float4 *__restrict__ c_tlo, float4 *__restrict__ c_thi) {
  if (info->cells_overflow) return;
  const int n_cells = info->n_cells;
  for (int c = blockIdx.x * blockDim.x + threadIdx.x; c < n_cells; c += gridDim.x * blockDim.x)
    moments_cell(c, (int)c_level[c], true, info, spos, c_link, c_first, c_count, c_cm, c_qa, c_qb, c_tlo, c_thi);
}

// internal cells of one level; its range comes from the level offsets on the device (no host round trip), so the
// launch is a fixed grid that strides over the level; levels 0..ltop are left to moments_top_kernel
__global__ void __launch_bounds__(128) moments_level_kernel(int level, const DevInfo *__restrict__ info,
                                                            const float4 *__restrict__ spos,
                                                            const uint2 *__restrict__ c_link,
                                                            const uint32_t *__restrict__ c_first,
                                                            uint32_t *__restrict__ c_count, float4 *__restrict__ c_cm,
                                                            float4 *__restrict__ c_qa, float4 *__restrict__ c_qb,
                                                            float4 *__restrict__ c_tlo, float4 *__restrict__ c_thi) {
  if (info->cells_overflow || level <= info->ltop) return;
  const int c0 = info->level_off[level], c1 = info->level_off[level + 1];
  for (int c = c0 + blockIdx.x * blockDim.x + threadIdx.x; c < c1; c += gridDim.x * blockDim.x)
    moments_cell(c, level, false, info, spos, c_link, c_first, c_count, c_cm, c_qa, c_qb, c_tlo, c_thi);
}

// internal cells of the top levels ltop .. 0 (few cells): one block, a block barrier between levels
__global__ void __launch_bounds__(256) moments_top_kernel(const DevInfo *__restrict__ info,
                                                          const float4 *__restrict__ spos, const uint2 *__restrict__ c_link,
                                                          const uint32_t *__restrict__ c_first,
                                                          uint32_t *__restrict__ c_count, float4 *__restrict__ c_cm,
                                                          float4 *__restrict__ c_qa, float4 *__restrict__ c_qb,
                                                          float4 *__restrict__ c_tlo, float4 *__restrict__ c_thi) {
  if (info->cells_overflow) return;
  for (int l = info->ltop; l >= 0; --l) {
    const int c0 = info->level_off[l], c1 = info->level_off[l + 1];
    for (int c = c0 + threadIdx.x; c < c1; c += blockDim.x)
      moments_cell(c, l, false, info, spos, c_link, c_first, c_count, c_cm, c_qa, c_qb, c_tlo, c_thi);
    __threadfence();
    __syncthreads();
  }
}

// ------------------------------------------------------------------------------------------
// host launchers
// ------------------------------------------------------------------------------------------
static inline int grid_for(tree_ctx *t, long long n, int threads, int per_sm) {
  long long need = (n + threads - 1) / threads;
  long long cap = (long long)t->sm_count * per_sm;
  return (int)(need < cap ? (need > 0 ? need : 1) : cap);
}

int run_pack_bbox(tree_ctx *t, const float *pos, const float *mass) {
  info_reset_kernel<<<1, 32, 0, t->stream>>>(t->d_info);
  BH_LAUNCH_CHECK("info_reset");
  bbox_kernel<true><<<grid_for(t, t->N, 256, 8), 256, 0, t->stream>>>(pos, mass, t->b.posm, t->N, t->d_info);
  BH_LAUNCH_CHECK("bbox_pack");
  return 0;
}

int run_kick_drift_bbox(tree_ctx *t, float dt) {
  info_reset_kernel<<<1, 32, 0, t->stream>>>(t->d_info);
  BH_LAUNCH_CHECK("info_reset");
  kick_drift_bbox_kernel<<<grid_for(t, t->N, 256, 8), 256, 0, t->stream>>>(t->b.spos, t->b.svel, t->b.sacc, t->N, 0.5f * dt,
                                                                            dt, t->d_info);
  BH_LAUNCH_CHECK("kick_drift_bbox");
  return 0;
}

int run_keys(tree_ctx *t, const float4 *xyzm) {
  grid_kernel<<<1, 32, 0, t->stream>>>(t->d_info);
  BH_LAUNCH_CHECK("grid");
  // the sort's first pass takes the identity as payload: no index array is written here
  keys_kernel<<<grid_for(t, t->N, 256, 8), 256, 0, t->stream>>>(
      xyzm, t->N, t->d_info, reinterpret_cast<const uint16_t *>(t->d_hlut + HLUT3_OFFSET), t->b.key[0], nullptr);
  BH_LAUNCH_CHECK("keys");
  return 0;
}

// The eight passes over `bound` keys starting in buffer `start` of key[] / idx[].  n_dev: the real count on the device
// (<= bound), or nullptr.  explicit_payload: idx[start] holds the payload (otherwise the first pass takes the identity).
static int sort_passes(tree_ctx *t, int start, long long bound, const unsigned *n_dev, bool explicit_payload) {
  if (!t->sort_attr_set) {  // per context: function attributes are per device
    BH_CUDA(cudaFuncSetAttribute(sort_onesweep_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(OsSmem)));
    BH_CUDA(cudaFuncSetAttribute(sort_onesweep_kernel, cudaFuncAttributePreferredSharedMemoryCarveout, 100));
    t->sort_attr_set = true;
  }
  const unsigned ntiles = (unsigned)((bound + OS_TILE - 1) / OS_TILE);
  uint32_t *ghist = t->b.sort_hist, *ticket = t->b.sort_hist + 8 * RADIX;
  BH_CUDA(cudaMemsetAsync(ghist, 0, 8 * RADIX * sizeof(uint32_t), t->stream));
  const long long hwant = (bound + 256 * 16 - 1) / (256 * 16), hcap = (long long)t->sm_count * 8;
  sort_hist8_kernel<<<(unsigned)(hwant < hcap ? hwant : hcap), 256, 0, t->stream>>>(t->b.key[start], bound, n_dev, ghist);
  BH_LAUNCH_CHECK("sort_hist8");
  sort_scan8_kernel<<<8, RADIX, 0, t->stream>>>(ghist, ticket);
  BH_LAUNCH_CHECK("sort_scan8");
  int cur = start;
  for (int pass = 0; pass < 8; ++pass) {
    const unsigned long long epoch = (++t->sort_epoch) & 0x3fffffffull;
    if (epoch == 0) {  // wrapped: old words could alias the new epoch
      BH_CUDA(cudaMemsetAsync(t->b.sort_status, 0, (size_t)t->sort_status_cap * sizeof(unsigned long long), t->stream));
      ++t->sort_epoch;
    }
    sort_onesweep_kernel<<<ntiles, OS_THREADS, sizeof(OsSmem), t->stream>>>(
        t->b.key[cur], (pass == 0 && !explicit_payload) ? nullptr : t->b.idx[cur], t->b.key[cur ^ 1], t->b.idx[cur ^ 1],
        ghist + pass * RADIX, ticket + pass, t->b.sort_status, t->sort_epoch & 0x3fffffffull, 8 * pass, bound, n_dev);
    BH_LAUNCH_CHECK("sort_onesweep");
    cur ^= 1;
  }
  t->sorted = cur;
  t->slot_of_valid = false;  // the passes used both key buffers, and the order is about to change
  return 0;
}

int run_sort(tree_ctx *t) {
  BH_TRY_RC(sort_passes(t, 0, t->N, nullptr, false));
  t->b.skey = t->b.key[t->sorted];
  t->b.sperm = t->b.idx[t->sorted];
  return 0;
}

// ------------------------------------------------------------------------------------------
// Sharded step: the sort is cut by KEY RANGE.  The keys found at the slot boundaries N r / world of
// the previous sorted order are splitters every rank holds; rank r takes the particles whose NEW key lies in
// [split[r], split[r+1]) -- its own slice of the previous order plus the few neighbours that crossed a boundary
// (contiguous pieces of the PH curve) -- sorts that bucket alone and stores the sorted (key, previous
// slot) run at the bucket's offset into every rank's xkey / xperm (peer stores).  After the caller's barrier all ranks
// hold the complete sorted arrays.  Equal keys all fall into one bucket; their order inside it is left to
// permute_step_kernel, which ranks ties by caller index anyway, so the compaction need not be stable.
// ------------------------------------------------------------------------------------------
__global__ void save_splitters_kernel(const uint64_t *__restrict__ skey, long long N, int world, DevInfo *info) {
  const int r = threadIdx.x;
  if (r < world) info->split[r] = r == 0 ? 0ull : skey[(N * r) / world];
}

__global__ void bucket_reset_kernel(DevInfo *info) {
  if (threadIdx.x < TREE_SHARD_MAX_WORLD) info->bucket_cnt[threadIdx.x] = 0u;
  if (threadIdx.x == 0) info->bucket_fill = 0u;
}

// counts every bucket (all ranks arrive at the same counts) and compacts this rank's bucket: (key, slot)
__global__ void __launch_bounds__(256) bucket_kernel(const uint64_t *__restrict__ key, long long N, int rank, int world,
                                                     DevInfo *info, uint64_t *__restrict__ out_key,
                                                     uint32_t *__restrict__ out_slot) {
  __shared__ unsigned long long sp[TREE_SHARD_MAX_WORLD];
  __shared__ unsigned cnt[TREE_SHARD_MAX_WORLD];
  if (threadIdx.x < TREE_SHARD_MAX_WORLD) {
    sp[threadIdx.x] = threadIdx.x < world ? info->split[threadIdx.x] : ~0ull;
    cnt[threadIdx.x] = 0u;
  }
  __syncthreads();
  const int lane = threadIdx.x & 31;
  for (long long base = (long long)blockIdx.x * blockDim.x; base < N; base += (long long)gridDim.x * blockDim.x) {
    const long long i = base + threadIdx.x;
    const bool valid = i < N;
    unsigned long long k = 0;
    int b = -1;
    if (valid) {
      k = key[i];
      b = 0;
      for (int r = 1; r < world; ++r) b += k >= sp[r];  // splitters are non-decreasing: b = last r with split[r] <= k
    }
    const unsigned same = __match_any_sync(0xffffffffu, b);  // neighbours on the curve share a bucket: one add per warp
    if (valid && lane == __ffs(same) - 1) atomicAdd(&cnt[b], (unsigned)__popc(same));
    const bool mine = b == rank;
    const unsigned m = __ballot_sync(0xffffffffu, mine);
    if (m) {
      unsigned at = 0;
      if (lane == __ffs(m) - 1) at = atomicAdd(&info->bucket_fill, (unsigned)__popc(m));
      at = __shfl_sync(0xffffffffu, at, __ffs(m) - 1);
      if (mine) {
        const unsigned dst = at + __popc(m & ((1u << lane) - 1u));
        out_key[dst] = k;
        out_slot[dst] = (uint32_t)i;
      }
    }
  }
  __syncthreads();
  if (threadIdx.x < world && cnt[threadIdx.x]) atomicAdd(&info->bucket_cnt[threadIdx.x], cnt[threadIdx.x]);
}

struct XDest { uint64_t *key[TREE_SHARD_MAX_WORLD]; uint32_t *perm[TREE_SHARD_MAX_WORLD]; int n; };

// the sorted bucket to its place in every rank's sorted arrays (own copy included)
__global__ void __launch_bounds__(256) bucket_store_kernel(const uint64_t *__restrict__ skey, const uint32_t *__restrict__ sperm,
                                                           int rank, const DevInfo *__restrict__ info, const XDest D) {
  const unsigned n = info->bucket_cnt[rank];
  unsigned off = 0;
  for (int r = 0; r < rank; ++r) off += info->bucket_cnt[r];
  for (unsigned i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
    const uint64_t k = skey[i];
    const uint32_t p = sperm[i];
    for (int q = 0; q < D.n; ++q) { D.key[q][off + i] = k; D.perm[q][off + i] = p; }
  }
}

int run_save_splitters(tree_ctx *t) {
  save_splitters_kernel<<<1, 32, 0, t->stream>>>(t->b.skey, t->N, t->shard_world, t->d_info);
  BH_LAUNCH_CHECK("save_splitters");
  t->split_valid = true;
  return 0;
}

int run_sort_bucket(tree_ctx *t) {
  bucket_reset_kernel<<<1, 32, 0, t->stream>>>(t->d_info);
  BH_LAUNCH_CHECK("bucket_reset");
  // new keys of all N are in key[0]; the bucket is compacted into key[1] / idx[1] and sorted from there
  bucket_kernel<<<grid_for(t, t->N, 256, 8), 256, 0, t->stream>>>(t->b.key[0], t->N, t->shard_rank, t->shard_world, t->d_info,
                                                                  t->b.key[1], t->b.idx[1]);
  BH_LAUNCH_CHECK("bucket");
  // the bucket's size is known on the device only: the grids cover all N, tiles past the end leave at once
  BH_TRY_RC(sort_passes(t, 1, t->N, &t->d_info->bucket_cnt[t->shard_rank], true));
  XDest D;
  D.n = 0;
  for (int r = 0; r < t->shard_world; ++r) {
    void *base = r == t->shard_rank ? t->b.shard_slab : t->peer_base[r];
    shard_xviews(t, base, &D.key[D.n], &D.perm[D.n]);
    ++D.n;
  }
  bucket_store_kernel<<<grid_for(t, (t->N + t->shard_world - 1) / t->shard_world, 256, 8), 256, 0, t->stream>>>(
      t->b.key[t->sorted], t->b.idx[t->sorted], t->shard_rank, t->d_info, D);
  BH_LAUNCH_CHECK("bucket_store");
  t->b.skey = t->b.xkey;
  t->b.sperm = t->b.xperm;
  return 0;
}

int run_permute_build(tree_ctx *t) {
  permute_build_kernel<<<(unsigned)((t->N + 255) / 256), 256, 0, t->stream>>>(t->b.posm, t->b.sperm, t->b.spos,
                                                                             t->b.order, t->N);
  BH_LAUNCH_CHECK("permute_build");
  return 0;
}

int run_permute_step(tree_ctx *t) {
  const int nxt = t->cur ^ 1;
  permute_step_kernel<<<(unsigned)((t->N + 255) / 256), 256, 0, t->stream>>>(
      t->b.skey, t->b.sperm, t->b.spos, t->b.svel, t->b.order, t->b.spos2[nxt], t->b.svel2[nxt],
      t->b.order2[nxt], t->rel_on && t->amag_valid ? t->b.amag2[t->cur] : nullptr, t->b.amag2[nxt], t->N);
  BH_LAUNCH_CHECK("permute_step");
  t->cur = nxt;
  t->b.spos = t->b.spos2[nxt]; t->b.svel = t->b.svel2[nxt]; t->b.order = t->b.order2[nxt];
  return 0;
}

// The cell count of the last asynchronous rebuild, if its read-back has arrived (never waits).
void poll_cells(tree_ctx *t) {
  if (!t->async_pending) return;
  if (cudaEventQuery(t->ev_async) != cudaSuccess) { cudaGetLastError(); return; }
  t->async_pending = false;
  if (t->h_async->n_cells > 0) t->n_cells = t->h_async->n_cells;
}

// !async (tree_build): one read-back of the cell count sizes the cell arrays exactly.
// async (tree_leapfrog): no host round trip.  The arrays hold cell_cap cells; the kernels may use
// cells_bound = min(cell_cap, latest known count + 1/8 + 1024) of them (the count changes by a fraction of a per cent
// per step), the device checks the real count against it (tree_offsets_kernel) and the count travels back
// asynchronously for the next step (poll_cells).
int run_tree(tree_ctx *t, bool async) {
  const int ntiles = (int)((t->N + TREE_THREADS - 1) / TREE_THREADS);
  const uint64_t *skey = t->b.skey;
  tree_levels_kernel<<<ntiles, TREE_THREADS, 0, t->stream>>>(skey, t->N, t->leaf, ntiles, t->b.lv, t->b.scan_tmp);
  BH_LAUNCH_CHECK("tree_levels");
  uint32_t *total = t->b.scan_blk + (t->scan_cap / SCAN_TILE + 8);  // spare slot behind the block sums
  int rc = device_excl_scan(t, t->b.scan_tmp, (long long)NLEVELS * ntiles, total);
  if (rc) return rc;
  if (async) {
    poll_cells(t);
    const long long want = t->n_cells + t->n_cells / 8 + 1024;
    t->cells_bound = want < t->cell_cap ? want : t->cell_cap;
  } else {
    t->cells_bound = 1ll << 28;  // checked on the host below
  }
  tree_offsets_kernel<<<1, 32, 0, t->stream>>>(t->b.scan_tmp, ntiles, total, t->cells_bound, t->d_info);
  BH_LAUNCH_CHECK("tree_offsets");
  if (async) {
    if (!t->async_pending) {  // the previous read-back has been consumed: start the next one
      BH_CUDA(cudaMemcpyAsync(t->h_async, t->d_info, sizeof(DevInfo), cudaMemcpyDeviceToHost, t->stream));
      BH_CUDA(cudaEventRecord(t->ev_async, t->stream));
      t->async_pending = true;
    }
  } else {
    BH_CUDA(cudaMemcpyAsync(t->h_info, t->d_info, sizeof(DevInfo), cudaMemcpyDeviceToHost, t->stream));
    BH_CUDA(cudaStreamSynchronize(t->stream));
    if (t->h_info->nonfinite) {  // reported now, not again later
      t->h_info->nonfinite_sticky = 0;
      cudaMemsetAsync(&t->d_info->nonfinite_sticky, 0, sizeof(unsigned), t->stream);
      return set_err(t, TREE_ERR_NONFINITE, "non-finite position or mass");
    }
    BH_TRY_RC(check_sticky(t));  // errors of earlier asynchronous passes surface here at the latest
    const long long nc = t->h_info->level_off[NLEVELS];
    if (nc <= 0 || nc >= (1ll << 28)) return set_err(t, TREE_ERR_ARG, "cell count out of range (needs < 2^28 cells)");
    rc = ensure_cells(t, nc);
    if (rc) return rc;
    t->n_cells = nc;
    t->cells_bound = nc;
    t->async_pending = false;
  }
  tree_emit_kernel<<<ntiles, TREE_THREADS, 0, t->stream>>>(t->b.lv, t->N, ntiles, t->b.scan_tmp, t->b.c_level,
                                                           t->b.c_first, t->b.c_count, t->b.c_fcall, t->d_info);
  BH_LAUNCH_CHECK("tree_emit");
  tree_link_kernel<<<(unsigned)((t->cells_bound + 255) / 256), 256, 0, t->stream>>>(t->d_info, t->b.c_first, t->b.c_count,
                                                                                    t->b.c_fcall, t->b.c_link);
  BH_LAUNCH_CHECK("tree_link");
  return 0;
}

int run_groups_moments(tree_ctx *t) {
  const long long thr = t->n_groups * 32;
  groups_kernel<<<(unsigned)((thr + 255) / 256), 256, 0, t->stream>>>(t->b.spos, t->N, t->group, t->n_groups, t->b.gbox);
  BH_LAUNCH_CHECK("groups");
  float4 *tlo = t->mac == TREE_MAC_BMAX ? t->b.c_tlo : nullptr, *thi = t->mac == TREE_MAC_BMAX ? t->b.c_thi : nullptr;
  // all grids below are sized from cells_bound; the kernels read the cell count and the level ranges on the device
  moments_leaf_kernel<<<grid_for(t, t->cells_bound, 128, 64), 128, 0, t->stream>>>(
      t->d_info, t->b.spos, t->b.c_link, t->b.c_level, t->b.c_first, t->b.c_count, t->b.c_cm, t->b.c_qa, t->b.c_qb, tlo, thi);
  BH_LAUNCH_CHECK("moments_leaf");
  for (int l = MAX_LEVEL; l >= 1; --l) {  // level 0 (the root) always belongs to the top block
    long long most = t->cells_bound;      // a level holds at most 8^l cells
    if (l < 9 && (1ll << (3 * l)) < most) most = 1ll << (3 * l);
    moments_level_kernel<<<grid_for(t, most, 128, 16), 128, 0, t->stream>>>(l, t->d_info, t->b.spos, t->b.c_link, t->b.c_first,
                                                                           t->b.c_count, t->b.c_cm, t->b.c_qa, t->b.c_qb, tlo, thi);
    BH_LAUNCH_CHECK("moments_level");
  }
  moments_top_kernel<<<1, 256, 0, t->stream>>>(t->d_info, t->b.spos, t->b.c_link, t->b.c_first, t->b.c_count, t->b.c_cm,
                                               t->b.c_qa, t->b.c_qb, tlo, thi);
  BH_LAUNCH_CHECK("moments_top");
  return 0;
}

// Hilbert state table from the Gray-code / rotation recurrence (T3), state = e*3 + d.
void build_hilbert_lut(uint8_t out[24 * 8]) {
  auto rot_r = [](unsigned x, unsigned k) { k %= 3; return ((x >> k) | (x << (3 - k))) & 7u; };
  auto rot_l = [](unsigned x, unsigned k) { k %= 3; return ((x << k) | (x >> (3 - k))) & 7u; };
  auto ones_tail = [](unsigned i) { unsigned n = 0; for (; i & 1u; i >>= 1) ++n; return n; };
  for (unsigned e = 0; e < 8; ++e)
    for (unsigned d = 0; d < 3; ++d)
      for (unsigned l = 0; l < 8; ++l) {
        unsigned g = rot_r(l ^ e, d + 1);
        unsigned w = g;  // inverse Gray code on 3 bits
        w ^= w >> 1;
        w ^= w >> 2;
        w &= 7u;
        unsigned ent = 0, dir = 0;
        if (w) {
          unsigned b = 2u * ((w - 1u) >> 1);
          ent = b ^ (b >> 1);
          dir = ((w & 1u) ? ones_tail(w) : ones_tail(w - 1u)) % 3u;
        }
        unsigned e2 = e ^ rot_l(ent, d + 1);
        unsigned d2 = (d + dir + 1u) % 3u;
        out[(e * 3 + d) * 8 + l] = (uint8_t)(w | ((e2 * 3 + d2) << 3));
      }
}

// Three levels per look-up (keys_kernel): entry [state][z3 y3 x3] = three digits, most significant first, | next state << 9.
void build_hilbert_lut3(const uint8_t lut[24 * 8], uint16_t out[HLUT3_ENTRIES]) {
  for (unsigned e = 0; e < (unsigned)HLUT3_ENTRIES; ++e) {
    const unsigned st = e >> 9, zt = (e >> 6) & 7u, yt = (e >> 3) & 7u, xt = e & 7u;
    // octant digit of a level = bits z y x of that level
    const unsigned o1 = ((zt >> 2) & 1u) << 2 | ((yt >> 2) & 1u) << 1 | ((xt >> 2) & 1u);
    const unsigned o2 = ((zt >> 1) & 1u) << 2 | ((yt >> 1) & 1u) << 1 | ((xt >> 1) & 1u);
    const unsigned o3 = (zt & 1u) << 2 | (yt & 1u) << 1 | (xt & 1u);
    const unsigned v1 = lut[st * 8 + o1], v2 = lut[(v1 >> 3) * 8 + o2], v3 = lut[(v2 >> 3) * 8 + o3];
    out[e] = (uint16_t)(((v1 & 7u) << 6) | ((v2 & 7u) << 3) | (v3 & 7u) | ((v3 >> 3) << 9));
  }
}

}  // namespace bh
