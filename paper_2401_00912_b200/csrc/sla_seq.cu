// sla_seq.cu -- sequence preparation: voxel coordinates -> window key -> window-sorted
// order -> gathered rows.  "These voxels are ordered based on their window coordinates, ensuring that voxels
// from the same window form a sub-matrix in contiguous memory"; windows are S_h x S_w cells of
// the ground plane.  Integer and byte work only; every result is unique, hence bit-exact
// (reading A16: the order inside a window is the input order, i.e. the sort is stable).
//
// The sort is a least-significant-digit radix sort, 8 bits per pass, ceil(bits(W) / 8) passes (two for the
// 3042 windows of a Waymo-like batch).  One pass is three kernels:
//   hist     a warp owns a tile of 512 consecutive keys and counts its digits            cnt[tile][digit]
//   scan     one block turns the counts into start positions in digit-major order        pre[tile][digit]
//   scatter  the warp walks its tile again 32 keys at a time, in order; match_any groups the lanes of equal
//            digit, a lane's rank in its group is its place behind the keys the warp already placed
// Equal digits keep their order inside a warp step (rank by lane), across the steps of a tile (running
// start position) and across tiles (scan order), so every pass is stable and so is the whole sort.
#include "sla_internal.cuh"

namespace sla {
namespace {

constexpr int kDigitBits = 8, kBins = 1 << kDigitBits;
constexpr int kTileSteps = 16, kTile = 32 * kTileSteps;   // keys per warp
constexpr int kSortWarps = 4;                            // warps (tiles) per block
constexpr int kScanGroups = 4;                           // scan block = kScanGroups x kBins threads

__global__ void __launch_bounds__(256)
sla_window_key_kernel(const int4* __restrict__ coords, int N, int batch, int grid_h, int grid_w, int S_h,
                      int S_w, int nwy, int nwx, int W, int32_t* __restrict__ key) {
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

__global__ void __launch_bounds__(32 * kSortWarps)
sla_sort_hist_kernel(const int32_t* __restrict__ key_in, int N, int shift, int T, uint32_t* __restrict__ cnt) {
  __shared__ uint32_t h[kSortWarps][kBins];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int t = blockIdx.x * kSortWarps + warp;
  if (t >= T) return;
#pragma unroll
  for (int j = 0; j < kBins / 32; ++j) h[warp][lane + 32 * j] = 0;
  __syncwarp();
  const long long base = (long long)t * kTile;
  int key[kTileSteps];
#pragma unroll
  for (int s = 0; s < kTileSteps; ++s) {
    const long long i = base + s * 32 + lane;
    key[s] = i < N ? __ldg(key_in + i) : 0;
  }
#pragma unroll
  for (int s = 0; s < kTileSteps; ++s) {
    const bool valid = base + s * 32 + lane < N;
    const int d = digit_of(key[s], shift, valid);
    const unsigned grp = __match_any_sync(0xffffffffu, d);
    if (valid && lane == __ffs(grp) - 1) h[warp][d] += __popc(grp);   // one writer per digit and step
    __syncwarp();
  }
#pragma unroll
  for (int j = 0; j < kBins / 32; ++j) cnt[(size_t)t * kBins + lane + 32 * j] = h[warp][lane + 32 * j];
}

// pre[t][d] = #keys with a smaller digit + #keys with digit d in tiles before t.  Thread (g, d) owns digit d
// of the g-th quarter of the tiles; consecutive threads read consecutive digits, so the walks are coalesced.
__global__ void __launch_bounds__(kScanGroups * kBins)
sla_sort_scan_kernel(uint32_t* __restrict__ cnt, int T) {
  __shared__ uint32_t part[kScanGroups][kBins];
  __shared__ uint32_t digit_base[kBins];
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
  if (threadIdx.x < 32) {                                 // exclusive scan of the 256 digit totals by one warp
    uint32_t v[kBins / 32], run = 0;
#pragma unroll
    for (int j = 0; j < kBins / 32; ++j) { v[j] = digit_base[threadIdx.x * (kBins / 32) + j]; run += v[j]; }
    uint32_t inc = run;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t up = __shfl_up_sync(0xffffffffu, inc, o);
      if ((int)threadIdx.x >= o) inc += up;
    }
    uint32_t ex = inc - run;
#pragma unroll
    for (int j = 0; j < kBins / 32; ++j) { digit_base[threadIdx.x * (kBins / 32) + j] = ex; ex += v[j]; }
  }
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

template <bool FIRST>
__global__ void __launch_bounds__(32 * kSortWarps)
sla_sort_scatter_kernel(const int32_t* __restrict__ key_in, const int32_t* __restrict__ val_in, int N, int shift,
                        int T, const uint32_t* __restrict__ pre, int32_t* __restrict__ key_out,
                        int32_t* __restrict__ val_out) {
  __shared__ uint32_t start[kSortWarps][kBins];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int t = blockIdx.x * kSortWarps + warp;
  if (t >= T) return;
#pragma unroll
  for (int j = 0; j < kBins / 32; ++j) start[warp][lane + 32 * j] = __ldg(pre + (size_t)t * kBins + lane + 32 * j);
  const long long base = (long long)t * kTile;
  int key[kTileSteps], val[kTileSteps];
#pragma unroll
  for (int s = 0; s < kTileSteps; ++s) {
    const long long i = base + s * 32 + lane;
    key[s] = i < N ? __ldg(key_in + i) : 0;
    val[s] = FIRST ? (int)i : (i < N ? __ldg(val_in + i) : 0);   // first pass: the value is the input position
  }
  __syncwarp();
  const unsigned below = (1u << lane) - 1u;
#pragma unroll
  for (int s = 0; s < kTileSteps; ++s) {
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

// dst[j] = src[perm[j]] (gather) or dst[perm[j]] = src[j] (scatter), rows of `vpr` vectors of type V.  A row
// whose perm entry lies outside [0, N) is skipped, so a bad permutation cannot reach outside the buffers.
template <typename V, bool SCATTER>
__global__ void __launch_bounds__(256)
sla_permute_rows_kernel(const V* __restrict__ src, const int32_t* __restrict__ perm, long long N, int vpr,
                        V* __restrict__ dst) {
  const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long row = idx / vpr;
  if (row >= N) return;
  const int col = (int)(idx - row * vpr);
  const long long p = __ldg(perm + row);
  if (p < 0 || p >= N) return;
  if (SCATTER) dst[p * vpr + col] = src[row * vpr + col];
  else         dst[row * vpr + col] = src[p * vpr + col];
}

}  // namespace

int sort_tiles(long long N) { return (int)((N + kTile - 1) / kTile); }

size_t sort_workspace_bytes(long long N) {
  const size_t n4 = ((size_t)N * 4 + 15) / 16 * 16;
  return 2 * n4 + (size_t)sort_tiles(N) * kBins * sizeof(uint32_t);
}

cudaError_t launch_window_keys(const int32_t* coords, int N, int batch, int grid_h, int grid_w, int S_h, int S_w,
                               int32_t* key, cudaStream_t st) {
  const int nwy = (grid_h + S_h - 1) / S_h, nwx = (grid_w + S_w - 1) / S_w;
  const unsigned blocks = (unsigned)(((long long)N + 255) / 256);
  sla_window_key_kernel<<<blocks, 256, 0, st>>>((const int4*)coords, N, batch, grid_h, grid_w, S_h, S_w, nwy, nwx,
                                                batch * nwy * nwx, key);
  return cudaGetLastError();
}

cudaError_t launch_sort_by_key(const int32_t* key, int N, int W, int32_t* perm, int32_t* key_sorted, void* ws,
                               cudaStream_t st) {
  const size_t n4 = ((size_t)N * 4 + 15) / 16 * 16;
  int32_t* key_tmp = (int32_t*)ws;
  int32_t* val_tmp = (int32_t*)((char*)ws + n4);
  uint32_t* cnt = (uint32_t*)((char*)ws + 2 * n4);
  const int T = sort_tiles(N);
  int bits = 0;
  while (bits < 31 && (W >> bits) != 0) ++bits;           // keys lie in [0, W]
  const int passes = bits == 0 ? 1 : (bits + kDigitBits - 1) / kDigitBits;
  const unsigned blocks = (unsigned)((T + kSortWarps - 1) / kSortWarps);
  const int32_t* kin = key;
  const int32_t* vin = nullptr;
  for (int p = 0; p < passes; ++p) {
    const bool to_user = ((passes - 1 - p) & 1) == 0;      // ping-pong so that the last pass lands in the outputs
    int32_t* kout = to_user ? key_sorted : key_tmp;
    int32_t* vout = to_user ? perm : val_tmp;
    const int shift = p * kDigitBits;
    sla_sort_hist_kernel<<<blocks, 32 * kSortWarps, 0, st>>>(kin, N, shift, T, cnt);
    sla_sort_scan_kernel<<<1, kScanGroups * kBins, 0, st>>>(cnt, T);
    if (p == 0) sla_sort_scatter_kernel<true><<<blocks, 32 * kSortWarps, 0, st>>>(kin, vin, N, shift, T, cnt, kout, vout);
    else        sla_sort_scatter_kernel<false><<<blocks, 32 * kSortWarps, 0, st>>>(kin, vin, N, shift, T, cnt, kout, vout);
    kin = kout;
    vin = vout;
  }
  return cudaGetLastError();
}

cudaError_t launch_permute_rows(const void* src, const int32_t* perm, long long N, size_t row_bytes, void* dst,
                                bool scatter, cudaStream_t st) {
  const bool wide = row_bytes % 16 == 0 && (((uintptr_t)src | (uintptr_t)dst) & 15u) == 0;
  const size_t vec = wide ? 16 : 4;
  const int vpr = (int)(row_bytes / vec);
  const unsigned long long total = (unsigned long long)N * (unsigned long long)vpr;
  const unsigned blocks = (unsigned)((total + 255) / 256);
  if (blocks == 0) return cudaSuccess;
  if (wide) {
    if (scatter) sla_permute_rows_kernel<uint4, true><<<blocks, 256, 0, st>>>((const uint4*)src, perm, N, vpr, (uint4*)dst);
    else         sla_permute_rows_kernel<uint4, false><<<blocks, 256, 0, st>>>((const uint4*)src, perm, N, vpr, (uint4*)dst);
  } else {
    if (scatter) sla_permute_rows_kernel<uint32_t, true><<<blocks, 256, 0, st>>>((const uint32_t*)src, perm, N, vpr, (uint32_t*)dst);
    else         sla_permute_rows_kernel<uint32_t, false><<<blocks, 256, 0, st>>>((const uint32_t*)src, perm, N, vpr, (uint32_t*)dst);
  }
  return cudaGetLastError();
}

}  // namespace sla
