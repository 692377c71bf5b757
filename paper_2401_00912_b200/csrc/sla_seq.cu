// sla_seq.cu -- sequence preparation: voxel coordinates -> window key -> window-sorted
// order -> gathered rows.  "These voxels are ordered based on their window coordinates, ensuring that voxels
// from the same window form a sub-matrix in contiguous memory"; windows are S_h x S_w cells of
// the ground plane.  Integer and byte work only; every result is unique, hence bit-exact
// (reading A16: the order inside a window is the input order, i.e. the sort is stable).
//
// The sort is a least-significant-digit radix sort, 8 bits per pass, ceil(bits(W) / 8) passes (two for the
// 3042 windows of a Waymo-like batch).  One pass is three kernels:
//   hist     a warp owns a tile of 128 (512 beyond 2^18 keys) consecutive keys and counts its digits; the 8 warps
//            of a block add their counts, so global memory sees one row per block                 cnt[block][digit]
//   scan     one block turns the counts into start positions in digit-major order        pre[block][digit]
//            (up to 128 blocks there is no such kernel: every scatter block sums the rows it needs itself)
//   scatter  the warps count again, take their start behind the warps before them, then walk their tile
//            32 keys at a time, in order; match_any groups the lanes of equal digit, a lane's rank in its
//            group is its place behind the keys the warp already placed
// Equal digits keep their order inside a warp step (rank by lane), across the steps of a tile (running
// start position), across the warps of a block and across blocks (scan order), so every pass is stable and
// so is the whole sort.  The kernels of a call form one chain of programmatic dependent launches: each lets
// its successor become resident at once and waits for its predecessor before it touches global memory.
#include "sla_internal.cuh"

namespace sla {
namespace {

constexpr int kDigitBits = 8, kBins = 1 << kDigitBits;
constexpr int kSortWarps = 8;                            // warps per block
// A warp walks STEPS x 32 keys in order, one dependent step after the other, so a short tile means a short
// kernel and more blocks to spread over the SMs; a long tile means fewer rows of counts for the one-block scan.
constexpr int kStepsSmall = 4, kStepsLarge = 16;
constexpr long long kSmallSortMax = 1 << 18;             // up to here: 4 steps (1024 keys per block)
constexpr int kOwnScanMax = 128;                         // up to this many blocks the scatter kernel scans for itself
constexpr int kScanGroups = 4;                           // scan block = kScanGroups x kBins threads
static_assert(32 * kSortWarps == kBins, "one thread per digit when the warps' counts are combined");

__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

__global__ void __launch_bounds__(256)
sla_window_key_kernel(const int4* __restrict__ coords, int N, int batch, int grid_h, int grid_w, int S_h,
                      int S_w, int nwy, int nwx, int W, int32_t* __restrict__ key) {
  pdl_launch_dependents();
  pdl_wait();
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  const int4 c = __ldg(coords + i);                      // (b, z, y, x); z takes no part
  const bool inside = (unsigned)c.x < (unsigned)batch && (unsigned)c.z < (unsigned)grid_h &&
                      (unsigned)c.w < (unsigned)grid_w;
  key[i] = inside ? (c.x * nwy + c.z / S_h) * nwx + c.w / S_w : W;
}

// digit of lane's key, or kBins for a lane past the end (a group of its own that is never counted)
__device__ __forceinline__ int digit_of(int key, int shift, bool valid) {
  return valid ? ((key >> shift) & (kBins - 1)) : kBins;
}

// The warp's 512 keys -> registers, and their digit counts -> h[0..255] (the warp's own row of shared memory).
template <int STEPS>
__device__ __forceinline__ void load_and_count(const int32_t* __restrict__ key_in, long long base, int N, int shift,
                                               int lane, int (&key)[STEPS], uint32_t* h) {
#pragma unroll
  for (int j = 0; j < kBins / 32; ++j) h[lane + 32 * j] = 0;
#pragma unroll
  for (int s = 0; s < STEPS; ++s) {
    const long long i = base + s * 32 + lane;
    key[s] = i < N ? key_in[i] : 0;                      // plain loads: the predecessor kernel wrote them
  }
  __syncwarp();
#pragma unroll
  for (int s = 0; s < STEPS; ++s) {
    const bool valid = base + s * 32 + lane < N;
    const int d = digit_of(key[s], shift, valid);
    const unsigned grp = __match_any_sync(0xffffffffu, d);
    if (valid && lane == __ffs(grp) - 1) h[d] += __popc(grp);   // one writer per digit and step
    __syncwarp();
  }
}

template <int STEPS>
__global__ void __launch_bounds__(32 * kSortWarps)
sla_sort_hist_kernel(const int32_t* __restrict__ key_in, int N, int shift, uint32_t* __restrict__ cnt) {
  __shared__ uint32_t h[kSortWarps][kBins];
  pdl_launch_dependents();
  pdl_wait();
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  int key[STEPS];
  load_and_count<STEPS>(key_in, ((long long)blockIdx.x * kSortWarps + warp) * (32 * STEPS), N, shift, lane, key, h[warp]);
  __syncthreads();
  uint32_t tot = 0;
#pragma unroll
  for (int w = 0; w < kSortWarps; ++w) tot += h[w][threadIdx.x];
  cnt[(size_t)blockIdx.x * kBins + threadIdx.x] = tot;
}

// exclusive scan of tot[0..255] in place, by the first warp of the block (the caller syncs before and after)
__device__ __forceinline__ void scan_digits(uint32_t* tot) {
  if (threadIdx.x < 32) {
    uint32_t v[kBins / 32], run = 0;
#pragma unroll
    for (int j = 0; j < kBins / 32; ++j) { v[j] = tot[threadIdx.x * (kBins / 32) + j]; run += v[j]; }
    uint32_t inc = run;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t up = __shfl_up_sync(0xffffffffu, inc, o);
      if ((int)threadIdx.x >= o) inc += up;
    }
    uint32_t ex = inc - run;
#pragma unroll
    for (int j = 0; j < kBins / 32; ++j) { tot[threadIdx.x * (kBins / 32) + j] = ex; ex += v[j]; }
  }
}

// pre[t][d] = #keys with a smaller digit + #keys with digit d in blocks before t.  Thread (g, d) owns digit d
// of the g-th quarter of the rows; consecutive threads read consecutive digits, so the walks are coalesced.
__global__ void __launch_bounds__(kScanGroups * kBins)
sla_sort_scan_kernel(uint32_t* __restrict__ cnt, int T) {
  __shared__ uint32_t part[kScanGroups][kBins];
  __shared__ uint32_t digit_base[kBins];
  pdl_launch_dependents();
  pdl_wait();
  const int g = threadIdx.x / kBins, d = threadIdx.x % kBins;
  const int per = (T + kScanGroups - 1) / kScanGroups;
  const int t0 = min(T, g * per), t1 = min(T, t0 + per);
  uint32_t sum = 0;
  for (int t = t0; t < t1; ++t) sum += cnt[(size_t)t * kBins + d];
  part[g][d] = sum;
  __syncthreads();
  if (g == 0) {
    uint32_t tot = 0;
#pragma unroll
    for (int j = 0; j < kScanGroups; ++j) tot += part[j][d];
    digit_base[d] = tot;
  }
  __syncthreads();
  scan_digits(digit_base);
  __syncthreads();
  uint32_t run = digit_base[d];
  for (int j = 0; j < g; ++j) run += part[j][d];
  for (int t = t0; t < t1; ++t) {
    const size_t at = (size_t)t * kBins + d;
    const uint32_t c = cnt[at];
    cnt[at] = run;
    run += c;
  }
}

// OWN_SCAN: `pre` holds the raw counts of all T blocks and every block works out its own start positions (few
// blocks: T rows of 1 KB out of L2 cost less than a kernel in between); else sla_sort_scan_kernel has run.
template <int STEPS, bool FIRST, bool OWN_SCAN>
__global__ void __launch_bounds__(32 * kSortWarps)
sla_sort_scatter_kernel(const int32_t* __restrict__ key_in, const int32_t* __restrict__ val_in, int N, int shift,
                        int T, const uint32_t* __restrict__ pre, int32_t* __restrict__ key_out,
                        int32_t* __restrict__ val_out) {
  __shared__ uint32_t start[kSortWarps][kBins];
  __shared__ uint32_t digit_base[kBins];
  pdl_launch_dependents();
  pdl_wait();
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const long long base = ((long long)blockIdx.x * kSortWarps + warp) * (32 * STEPS);
  int key[STEPS], val[STEPS];
  load_and_count<STEPS>(key_in, base, N, shift, lane, key, start[warp]);
#pragma unroll
  for (int s = 0; s < STEPS; ++s) {
    const long long i = base + s * 32 + lane;
    val[s] = FIRST ? (int)i : (i < N ? val_in[i] : 0);    // first pass: the value is the input position
  }
  uint32_t run;
  if (OWN_SCAN) {
    uint32_t before = 0, all = 0;                         // thread d: digit d in the blocks before this one / in all
    for (int t = 0; t < T; ++t) {
      const uint32_t c = pre[(size_t)t * kBins + threadIdx.x];
      all += c;
      if (t < (int)blockIdx.x) before += c;
    }
    digit_base[threadIdx.x] = all;
    __syncthreads();
    scan_digits(digit_base);
    __syncthreads();
    run = digit_base[threadIdx.x] + before;
  } else {
    run = pre[(size_t)blockIdx.x * kBins + threadIdx.x];
    __syncthreads();
  }
#pragma unroll
  for (int w = 0; w < kSortWarps; ++w) {                  // counts -> starts, warp by warp behind the block's start
    const uint32_t c = start[w][threadIdx.x];
    start[w][threadIdx.x] = run;
    run += c;
  }
  __syncthreads();
  const unsigned below = (1u << lane) - 1u;
#pragma unroll
  for (int s = 0; s < STEPS; ++s) {
    const bool valid = base + s * 32 + lane < N;
    const int d = digit_of(key[s], shift, valid);
    const unsigned grp = __match_any_sync(0xffffffffu, d);
    uint32_t pos = 0;
    if (valid) pos = start[warp][d] + __popc(grp & below);
    __syncwarp();
    if (valid && lane == __ffs(grp) - 1) start[warp][d] += __popc(grp);
    __syncwarp();
    if (valid) { key_out[pos] = key[s]; val_out[pos] = val[s]; }
  }
}

// ---- one scene: counting sort in one pass ------------------------------------------------------------------------------
// A single frame has W = 1521 windows (468 x 468 cells in 12 x 12 windows): the key itself is the only digit.  Two
// kernels instead of six (keys, 2 x (hist, scatter), offsets):
//   count   keys of a tile of 1024 voxels -> key[], their histogram over the W + 1 bins -> cnt[block][bin] (uint16)
//   place   every block sums the rows before it and all rows (thread = 8 consecutive bins = one 16-byte load per row),
//           scans the totals -- which ARE the window offsets: block 0 writes them --, ranks its keys warp by warp
//           and step by step as the radix scatter does (stable), and writes perm / key_sorted
constexpr int kSeqBins = 2048;                           // W + 1 <= kSeqBins
constexpr int kSeqSteps = 4;
constexpr int kSeqTile = 32 * kSortWarps * kSeqSteps;    // 1024 voxels per block
static_assert(kSeqBins == 8 * 32 * kSortWarps, "a thread owns 8 consecutive bins");

__global__ void __launch_bounds__(32 * kSortWarps)
sla_seq_count_kernel(const int4* __restrict__ coords, int N, int batch, int grid_h, int grid_w, int S_h, int S_w,
                     int nwy, int nwx, int W, int32_t* __restrict__ key, uint16_t* __restrict__ cnt) {
  __shared__ uint32_t h[kSeqBins];
  pdl_launch_dependents();
#pragma unroll
  for (int j = 0; j < kSeqBins / (32 * kSortWarps); ++j) h[threadIdx.x + j * 32 * kSortWarps] = 0;
  __syncthreads();
  pdl_wait();
  const long long base = (long long)blockIdx.x * kSeqTile;
#pragma unroll
  for (int s = 0; s < kSeqSteps; ++s) {
    const long long i = base + s * (32 * kSortWarps) + threadIdx.x;
    if (i < N) {
      const int4 c = __ldg(coords + i);                  // (b, z, y, x); z takes no part
      const bool inside = (unsigned)c.x < (unsigned)batch && (unsigned)c.z < (unsigned)grid_h &&
                          (unsigned)c.w < (unsigned)grid_w;
      const int kk = inside ? (c.x * nwy + c.z / S_h) * nwx + c.w / S_w : W;
      key[i] = kk;
      atomicAdd(&h[kk], 1u);
    }
  }
  __syncthreads();
  const uint32_t* m = h + 8 * threadIdx.x;               // counts <= 1024: 16 bits each
  reinterpret_cast<uint4*>(cnt + (size_t)blockIdx.x * kSeqBins)[threadIdx.x] =
      make_uint4(m[0] | (m[1] << 16), m[2] | (m[3] << 16), m[4] | (m[5] << 16), m[6] | (m[7] << 16));
}

__global__ void __launch_bounds__(32 * kSortWarps)
sla_seq_place_kernel(const int32_t* __restrict__ key_in, int N, int W, int T, const uint16_t* __restrict__ cnt,
                     int32_t* __restrict__ perm, int32_t* __restrict__ key_sorted, int32_t* __restrict__ off) {
  __shared__ __align__(16) uint16_t rel[kSortWarps][kSeqBins];   // per warp: count, then start behind the warps before
  __shared__ uint32_t basepos[kSeqBins];                         // start of this block's keys of a bin in the output
  __shared__ uint32_t warp_sum[kSortWarps];
  pdl_launch_dependents();
  {
    uint4* z = reinterpret_cast<uint4*>(&rel[0][0]);
#pragma unroll
    for (int j = 0; j < (int)(sizeof(rel) / 16) / (32 * kSortWarps); ++j)
      z[threadIdx.x + j * 32 * kSortWarps] = make_uint4(0, 0, 0, 0);
  }
  __syncthreads();
  pdl_wait();
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const long long base = (long long)blockIdx.x * kSeqTile + warp * (32 * kSeqSteps);
  int kk[kSeqSteps];
#pragma unroll
  for (int s = 0; s < kSeqSteps; ++s) {
    const long long i = base + s * 32 + lane;
    kk[s] = i < N ? key_in[i] : kSeqBins;                 // past the end: a group of its own that is never counted
  }
#pragma unroll
  for (int s = 0; s < kSeqSteps; ++s) {
    const unsigned grp = __match_any_sync(0xffffffffu, kk[s]);
    if (kk[s] < kSeqBins && lane == __ffs(grp) - 1) rel[warp][kk[s]] += (uint16_t)__popc(grp);
    __syncwarp();
  }
  // bins 8 tid .. 8 tid + 7: keys in the blocks before this one, and in all blocks
  uint32_t before[8], all[8];
#pragma unroll
  for (int j = 0; j < 8; ++j) before[j] = all[j] = 0;
  const uint4* rows = reinterpret_cast<const uint4*>(cnt) + threadIdx.x;
  auto add_row = [&](const uint4& r, uint32_t (&acc)[8]) {
    acc[0] += r.x & 0xffffu; acc[1] += r.x >> 16; acc[2] += r.y & 0xffffu; acc[3] += r.y >> 16;
    acc[4] += r.z & 0xffffu; acc[5] += r.z >> 16; acc[6] += r.w & 0xffffu; acc[7] += r.w >> 16;
  };
  constexpr int kRowsInFlight = 16;                      // the rows come out of L2 one latency per batch, not per row
  for (int t0 = 0; t0 < T; t0 += kRowsInFlight) {
    uint4 r[kRowsInFlight];
#pragma unroll
    for (int u = 0; u < kRowsInFlight; ++u)               // plain loads: the count kernel wrote them
      r[u] = t0 + u < T ? rows[(size_t)(t0 + u) * (kSeqBins / 8)] : make_uint4(0, 0, 0, 0);
#pragma unroll
    for (int u = 0; u < kRowsInFlight; ++u) {
      if (t0 + u < (int)blockIdx.x) add_row(r[u], before);
      else add_row(r[u], all);
    }
  }
  uint32_t mine = 0;
#pragma unroll
  for (int j = 0; j < 8; ++j) { all[j] += before[j]; mine += all[j]; }
  uint32_t inc = mine;                                   // block-wide exclusive scan of the bin totals
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const uint32_t up = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += up;
  }
  if (lane == 31) warp_sum[warp] = inc;
  __syncthreads();                                       // also: every warp's counts are in rel[][]
  uint32_t ex = inc - mine;
  for (int w = 0; w < warp; ++w) ex += warp_sum[w];
#pragma unroll
  for (int j = 0; j < 8; ++j) {
    const int d = 8 * threadIdx.x + j;
    if (blockIdx.x == 0 && d <= W) off[d] = (int32_t)ex;  // keys below d = first row of window d; off[W] = voxels inside
    basepos[d] = ex + before[j];
    ex += all[j];
  }
  {
    // counts -> starts behind the warps before, for this thread's 8 bins at once (packed 16-bit pairs: a pair of
    // counts sums to <= 1024, no carry between the halves)
    uint4 run = make_uint4(0, 0, 0, 0);
#pragma unroll
    for (int w = 0; w < kSortWarps; ++w) {
      uint4* at = reinterpret_cast<uint4*>(&rel[w][8 * threadIdx.x]);
      const uint4 c = *at;
      *at = run;
      run.x += c.x; run.y += c.y; run.z += c.z; run.w += c.w;
    }
  }
  __syncthreads();
  const unsigned below = (1u << lane) - 1u;
#pragma unroll
  for (int s = 0; s < kSeqSteps; ++s) {
    const bool valid = kk[s] < kSeqBins;
    const unsigned grp = __match_any_sync(0xffffffffu, kk[s]);
    uint32_t pos = 0;
    if (valid) pos = basepos[kk[s]] + rel[warp][kk[s]] + __popc(grp & below);
    __syncwarp();
    if (valid && lane == __ffs(grp) - 1) rel[warp][kk[s]] += (uint16_t)__popc(grp);
    __syncwarp();
    if (valid) { key_sorted[pos] = kk[s]; perm[pos] = (int32_t)(base + s * 32 + lane); }
  }
}

// dst[j] = src[perm[j]] (gather) or dst[perm[j]] = src[j] (scatter), rows of `vpr` vectors of type V.  A row
// whose perm entry lies outside [0, N) is skipped, so a bad permutation cannot reach outside the buffers.
// A thread moves kPermUnroll vectors, 256 apart, and has all its loads in flight before the first store.
constexpr int kPermUnroll = 4;
template <typename V, bool SCATTER>
__global__ void __launch_bounds__(256)
sla_permute_rows_kernel(const V* __restrict__ src, const int32_t* __restrict__ perm, long long N, int vpr, int shift,
                        V* __restrict__ dst) {
  pdl_launch_dependents();
  pdl_wait();
  const long long total = N * vpr;
  const long long first = (long long)blockIdx.x * (256 * kPermUnroll) + threadIdx.x;
  long long from[kPermUnroll], to[kPermUnroll];
  V x[kPermUnroll];
#pragma unroll
  for (int u = 0; u < kPermUnroll; ++u) {
    const long long idx = first + u * 256;
    from[u] = -1;
    if (idx < total) {
      // vectors per row is a power of two for the usual rows (256 or 512 bytes): a shift instead of a 64-bit division
      const long long row = shift >= 0 ? (idx >> shift) : idx / vpr;
      const int col = (int)(idx - row * vpr);
      const long long p = perm[row];
      if (p >= 0 && p < N) {
        from[u] = (SCATTER ? row : p) * vpr + col;
        to[u] = (SCATTER ? p : row) * vpr + col;
      }
    }
  }
#pragma unroll
  for (int u = 0; u < kPermUnroll; ++u)
    if (from[u] >= 0) x[u] = src[from[u]];
#pragma unroll
  for (int u = 0; u < kPermUnroll; ++u)
    if (from[u] >= 0) dst[to[u]] = x[u];
}

// One link of a chain of programmatic dependent launches (see the kernels: launch_dependents, then wait).
template <typename... KArgs, typename... Args>
cudaError_t launch_chained(void (*kernel)(KArgs...), unsigned blocks, unsigned threads, cudaStream_t st, Args... args) {
  cudaLaunchAttribute pdl[1];
  pdl[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  pdl[0].val.programmaticStreamSerializationAllowed = 1;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(blocks);
  cfg.blockDim = dim3(threads);
  cfg.stream = st;
  cfg.attrs = pdl;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

}  // namespace

static int sort_steps(long long N) { return N <= kSmallSortMax ? kStepsSmall : kStepsLarge; }
static int sort_blocks(long long N) {
  const long long tile = (long long)kSortWarps * 32 * sort_steps(N);
  return (int)((N + tile - 1) / tile);
}

template <int STEPS>
static cudaError_t sort_pass(const int32_t* kin, const int32_t* vin, int N, int shift, int T, uint32_t* cnt,
                             int32_t* kout, int32_t* vout, bool first, cudaStream_t st) {
  cudaError_t e = launch_chained(sla_sort_hist_kernel<STEPS>, T, 32 * kSortWarps, st, kin, N, shift, cnt);
  if (e != cudaSuccess) return e;
  if (T <= kOwnScanMax)
    return first ? launch_chained(sla_sort_scatter_kernel<STEPS, true, true>, T, 32 * kSortWarps, st, kin, vin, N, shift, T, cnt, kout, vout)
                 : launch_chained(sla_sort_scatter_kernel<STEPS, false, true>, T, 32 * kSortWarps, st, kin, vin, N, shift, T, cnt, kout, vout);
  e = launch_chained(sla_sort_scan_kernel, 1, kScanGroups * kBins, st, cnt, T);
  if (e != cudaSuccess) return e;
  return first ? launch_chained(sla_sort_scatter_kernel<STEPS, true, false>, T, 32 * kSortWarps, st, kin, vin, N, shift, T, cnt, kout, vout)
               : launch_chained(sla_sort_scatter_kernel<STEPS, false, false>, T, 32 * kSortWarps, st, kin, vin, N, shift, T, cnt, kout, vout);
}

size_t sort_workspace_bytes(long long N) {
  const size_t n4 = ((size_t)N * 4 + 15) / 16 * 16;
  return 2 * n4 + (size_t)sort_blocks(N) * kBins * sizeof(uint32_t);
}

cudaError_t launch_window_keys(const int32_t* coords, int N, int batch, int grid_h, int grid_w, int S_h, int S_w,
                               int32_t* key, cudaStream_t st) {
  const int nwy = (grid_h + S_h - 1) / S_h, nwx = (grid_w + S_w - 1) / S_w;
  const unsigned blocks = (unsigned)(((long long)N + 255) / 256);
  return launch_chained(sla_window_key_kernel, blocks, 256, st, (const int4*)coords, N, batch, grid_h, grid_w, S_h,
                        S_w, nwy, nwx, batch * nwy * nwx, key);
}

cudaError_t launch_sort_by_key(const int32_t* key, int N, int W, int32_t* perm, int32_t* key_sorted, void* ws,
                               cudaStream_t st) {
  const size_t n4 = ((size_t)N * 4 + 15) / 16 * 16;
  int32_t* key_tmp = (int32_t*)ws;
  int32_t* val_tmp = (int32_t*)((char*)ws + n4);
  uint32_t* cnt = (uint32_t*)((char*)ws + 2 * n4);
  const int T = sort_blocks(N);
  int bits = 0;
  while (bits < 31 && (W >> bits) != 0) ++bits;           // keys lie in [0, W]
  const int passes = bits == 0 ? 1 : (bits + kDigitBits - 1) / kDigitBits;
  const int32_t* kin = key;
  const int32_t* vin = nullptr;
  cudaError_t e = cudaSuccess;
  for (int p = 0; p < passes && e == cudaSuccess; ++p) {
    const bool to_user = ((passes - 1 - p) & 1) == 0;      // ping-pong so that the last pass lands in the outputs
    int32_t* kout = to_user ? key_sorted : key_tmp;
    int32_t* vout = to_user ? perm : val_tmp;
    const int shift = p * kDigitBits;
    e = sort_steps(N) == kStepsSmall ? sort_pass<kStepsSmall>(kin, vin, N, shift, T, cnt, kout, vout, p == 0, st)
                                     : sort_pass<kStepsLarge>(kin, vin, N, shift, T, cnt, kout, vout, p == 0, st);
    kin = kout;
    vin = vout;
  }
  return e;
}

// `scratch`: bytes available for the per-block counts
bool sequence_onepass_fits(long long N, long long W, size_t scratch) {
  if (N <= 0 || W + 1 > kSeqBins) return false;
  const size_t T = (size_t)((N + kSeqTile - 1) / kSeqTile);
  return T * kSeqBins * sizeof(uint16_t) <= scratch;
}

// cnt: ceil(N / 1024) rows of kSeqBins uint16 (4 bytes per voxel, 16-byte aligned)
cudaError_t launch_sequence_onepass(const int32_t* coords, int N, int batch, int grid_h, int grid_w, int S_h, int S_w,
                                    int32_t* key, void* cnt, int32_t* perm, int32_t* key_sorted, int32_t* off,
                                    cudaStream_t st) {
  const int nwy = (grid_h + S_h - 1) / S_h, nwx = (grid_w + S_w - 1) / S_w;
  const int W = batch * nwy * nwx;
  const int T = (int)(((long long)N + kSeqTile - 1) / kSeqTile);
  cudaError_t e = launch_chained(sla_seq_count_kernel, T, 32 * kSortWarps, st, (const int4*)coords, N, batch, grid_h,
                                 grid_w, S_h, S_w, nwy, nwx, W, key, (uint16_t*)cnt);
  if (e != cudaSuccess) return e;
  return launch_chained(sla_seq_place_kernel, T, 32 * kSortWarps, st, (const int32_t*)key, N, W, T,
                        (const uint16_t*)cnt, perm, key_sorted, off);
}

cudaError_t launch_permute_rows(const void* src, const int32_t* perm, long long N, size_t row_bytes, void* dst,
                                bool scatter, cudaStream_t st) {
  const bool wide = row_bytes % 16 == 0 && (((uintptr_t)src | (uintptr_t)dst) & 15u) == 0;
  const size_t vec = wide ? 16 : 4;
  const int vpr = (int)(row_bytes / vec);
  int shift = -1;                                          // log2(vpr) if vpr is a power of two
  for (int b = 0; b < 31; ++b)
    if (vpr == (1 << b)) shift = b;
  const unsigned long long total = (unsigned long long)N * (unsigned long long)vpr;
  const unsigned long long per_block = 256ull * kPermUnroll;
  const unsigned blocks = (unsigned)((total + per_block - 1) / per_block);
  if (blocks == 0) return cudaSuccess;
  if (wide)
    return scatter ? launch_chained(sla_permute_rows_kernel<uint4, true>, blocks, 256, st, (const uint4*)src, perm, N, vpr, shift, (uint4*)dst)
                   : launch_chained(sla_permute_rows_kernel<uint4, false>, blocks, 256, st, (const uint4*)src, perm, N, vpr, shift, (uint4*)dst);
  return scatter ? launch_chained(sla_permute_rows_kernel<uint32_t, true>, blocks, 256, st, (const uint32_t*)src, perm, N, vpr, shift, (uint32_t*)dst)
                 : launch_chained(sla_permute_rows_kernel<uint32_t, false>, blocks, 256, st, (const uint32_t*)src, perm, N, vpr, shift, (uint32_t*)dst);
}

}  // namespace sla
