// sla_cwi.cu -- Cross-Window Interaction (Eq. 4-7): the 4c input channels are split
// into four branches, depth-wise sparse convolutions with an (S_h+1)-tap kernel along y, an (S_w+1)-tap kernel along x
// and a 3x3x3 kernel, and an identity branch; outputs live on the input's voxels, a tap on an empty cell contributes
// nothing (reading A18).
//
// A gather: per voxel at most S_h + S_w + 29 neighbour look-ups and, for the few that exist, c channels of one branch
// (64 bytes at c = 32) out of L2.  No contraction, nothing for the tensor cores.  Three kernels, one chain of
// programmatic dependent launches:
//   fill     the dense index grid [batch, Z, H, W] (int32, caller's workspace) <- -1
//   scatter  grid[cell of voxel i] <- i
//   conv     one warp per voxel: the lanes look up all taps at once (lane t owns tap t, t+32, ..), the indices are
//            broadcast tap by tap, empty taps are skipped by the whole warp, lane l accumulates channels l, l+32, ..
//            of every branch in fp32 with the weights staged in shared memory as [tap][channel]; one rounding to the
//            I/O dtype; taps are added in index order, so the result is deterministic.
#include "sla_internal.cuh"

namespace sla {
namespace {

__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

__global__ void __launch_bounds__(256) sla_cwi_fill_kernel(uint4* __restrict__ p, size_t n16) {
  pdl_launch_dependents();
  pdl_wait();   // a previous call's conv kernel may still be reading the grid
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n16; i += (size_t)gridDim.x * blockDim.x)
    p[i] = make_uint4(0xFFFFFFFFu, 0xFFFFFFFFu, 0xFFFFFFFFu, 0xFFFFFFFFu);
}

struct Geom { int batch, gz, gh, gw; };

__device__ __forceinline__ long long cell_of(const Geom& g, int b, int z, int y, int x) {
  const bool inside = (unsigned)b < (unsigned)g.batch && (unsigned)z < (unsigned)g.gz && (unsigned)y < (unsigned)g.gh &&
                      (unsigned)x < (unsigned)g.gw;
  return inside ? (((long long)b * g.gz + z) * g.gh + y) * g.gw + x : -1;
}

__global__ void __launch_bounds__(256)
sla_cwi_scatter_kernel(const int4* __restrict__ coords, int N, Geom g, int32_t* __restrict__ grid) {
  pdl_launch_dependents();
  pdl_wait();
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  const int4 c = __ldg(coords + i);                      // (b, z, y, x)
  const long long cell = cell_of(g, c.x, c.y, c.z, c.w);
  if (cell >= 0) grid[cell] = (int)i;                    // a voxel outside the grid is seen by nobody
}

template <typename T> __device__ __forceinline__ float ld_elem(const T* p);
template <> __device__ __forceinline__ float ld_elem<float>(const float* p) { return __ldg(p); }
template <> __device__ __forceinline__ float ld_elem<__half>(const __half* p) { return __half2float(__ldg(p)); }
template <> __device__ __forceinline__ float ld_elem<__nv_bfloat16>(const __nv_bfloat16* p) { return __bfloat162float(__ldg(p)); }
template <typename T> __device__ __forceinline__ T to_elem(float v);
template <> __device__ __forceinline__ float to_elem<float>(float v) { return v; }
template <> __device__ __forceinline__ __half to_elem<__half>(float v) { return __float2half_rn(v); }
template <> __device__ __forceinline__ __nv_bfloat16 to_elem<__nv_bfloat16>(float v) { return __float2bfloat16_rn(v); }

constexpr int kCwiWarps = 16;

// CPL = channels of a branch per lane = ceil(c / 32); NS = 32-tap slots = ceil((S_h + S_w + 29) / 32)
template <typename T, int CPL, int NS>
__global__ void __launch_bounds__(32 * kCwiWarps)
sla_cwi_conv_kernel(const T* __restrict__ x, const int4* __restrict__ coords, int N, int C, Geom g, int S_h, int S_w,
                    const float* __restrict__ w_h, const float* __restrict__ w_w, const float* __restrict__ w_3,
                    const int32_t* __restrict__ grid, T* __restrict__ out) {
  extern __shared__ float s_w[];                         // [T_h + T_w + 27][c]: tap-major copies of the three weights
  pdl_launch_dependents();
  const int c = C >> 2;
  const int Th = S_h + 1, Tw = S_w + 1, Tall = Th + Tw + 27;
  // weights are the caller's constants, not a predecessor's output: staged before the dependency wait
  for (int i = threadIdx.x; i < Tall * c; i += blockDim.x) {
    const int t = i / c, ch = i - t * c;
    float v;
    if (t < Th) v = __ldg(w_h + ch * Th + t);
    else if (t < Th + Tw) v = __ldg(w_w + ch * Tw + (t - Th));
    else v = __ldg(w_3 + ch * 27 + (t - Th - Tw));
    s_w[i] = v;
  }
  pdl_wait();
  __syncthreads();
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  // the taps a lane owns (tap t = lane + 32 s) and their offsets do not depend on the voxel
  int tdz[NS], tdy[NS], tdx[NS], tdelta[NS];
#pragma unroll
  for (int s = 0; s < NS; ++s) {
    const int t = lane + 32 * s;
    int dz = 0, dy = 0, dx = 0;
    if (t < Th) dy = t - (S_h >> 1);
    else if (t < Th + Tw) dx = t - Th - (S_w >> 1);
    else if (t < Tall) { const int u = t - Th - Tw; dz = u / 9 - 1; dy = (u / 3) % 3 - 1; dx = u % 3 - 1; }
    else dz = 1 << 20;                                     // no such tap: always outside the grid
    tdz[s] = dz; tdy[s] = dy; tdx[s] = dx;
    tdelta[s] = (dz * g.gh + dy) * g.gw + dx;              // |.| < 2^31 cells
  }
  // bit masks of the taps of each branch inside each 32-tap slot
  unsigned bmask[3][NS];
#pragma unroll
  for (int s = 0; s < NS; ++s) {
    const int lo = 32 * s;
    auto range_mask = [&](int a, int b) -> unsigned {      // taps [a, b) intersected with [lo, lo + 32)
      const int x0 = max(a, lo) - lo, x1 = min(b, lo + 32) - lo;
      if (x1 <= x0) return 0u;
      return (x1 - x0 == 32) ? 0xffffffffu : (((1u << (x1 - x0)) - 1u) << x0);
    };
    bmask[0][s] = range_mask(0, Th);
    bmask[1][s] = range_mask(Th, Th + Tw);
    bmask[2][s] = range_mask(Th + Tw, Tall);
  }
  // the centre tap of every branch is the voxel itself: no look-up, no shuffle; taken out of the masks
  const int tc[3] = {S_h >> 1, Th + (S_w >> 1), Th + Tw + 13};
#pragma unroll
  for (int br = 0; br < 3; ++br)
#pragma unroll
    for (int s = 0; s < NS; ++s)
      if ((tc[br] >> 5) == s) bmask[br][s] &= ~(1u << (tc[br] & 31));
  // the grid cells of the taps this lane owns around voxel `me` -> idx[] (-1: no voxel there)
  auto lookups = [&](const int4& me, int (&idx)[NS]) -> bool {
    const bool me_in = (unsigned)me.x < (unsigned)g.batch && (unsigned)me.y < (unsigned)g.gz &&
                       (unsigned)me.z < (unsigned)g.gh && (unsigned)me.w < (unsigned)g.gw;
    const long long cell0 = (((long long)me.x * g.gz + me.y) * g.gh + me.z) * g.gw + me.w;
#pragma unroll
    for (int s = 0; s < NS; ++s) {
      const bool inside = me_in && (unsigned)(me.y + tdz[s]) < (unsigned)g.gz &&
                          (unsigned)(me.z + tdy[s]) < (unsigned)g.gh && (unsigned)(me.w + tdx[s]) < (unsigned)g.gw;
      idx[s] = inside ? grid[cell0 + tdelta[s]] : -1;
    }
    return me_in;
  };
  // Persistent warps (the weights are staged once per block, the tap set-up done once per warp), software-pipelined:
  // while voxel i is processed, the look-ups of the warp's next voxel and the coordinates of the one after are in flight.
  const long long stride = (long long)gridDim.x * kCwiWarps;
  long long i = (long long)blockIdx.x * kCwiWarps + warp;
  const int4 none = make_int4(-1, -1, -1, -1);             // outside every grid: all look-ups give -1 without a load
  int idx[NS];
  bool in_grid = lookups(i < N ? __ldg(coords + i) : none, idx);
  int4 me_next = (i + stride < N) ? __ldg(coords + i + stride) : none;
  for (; i < N; i += stride) {
    int idx_next[NS];
    const bool in_grid_next = lookups(me_next, idx_next);
    me_next = (i + 2 * stride < N) ? __ldg(coords + i + 2 * stride) : none;
    const T* xrow = x + (size_t)i * C;
    float acc[3][CPL];
#pragma unroll
    for (int br = 0; br < 3; ++br) {
#pragma unroll
      for (int k = 0; k < CPL; ++k) {                      // centre tap (a voxel off the grid gets zeros here)
        const int ch = lane + 32 * k;
        acc[br][k] = (in_grid && ch < c) ? s_w[tc[br] * c + ch] * ld_elem<T>(xrow + br * c + ch) : 0.f;
      }
      const T* xb = x + br * c;
#pragma unroll
      for (int s = 0; s < NS; ++s) {
        unsigned present = __ballot_sync(0xffffffffu, idx[s] >= 0) & bmask[br][s];   // this branch's taps that hit a voxel
        while (present) {                                                            // ascending: deterministic sums
          const int l = __ffs(present) - 1;
          present &= present - 1;
          const int j = __shfl_sync(0xffffffffu, idx[s], l);
          const T* row = xb + (size_t)j * C;
          const float* wt = s_w + (l + 32 * s) * c;
#pragma unroll
          for (int k = 0; k < CPL; ++k) {
            const int ch = lane + 32 * k;
            if (ch < c) acc[br][k] += wt[ch] * ld_elem<T>(row + ch);
          }
        }
      }
    }
    T* orow = out + (size_t)i * C;
#pragma unroll
    for (int k = 0; k < CPL; ++k) {
      const int ch = lane + 32 * k;
      if (ch < c) {
        orow[ch] = to_elem<T>(acc[0][k]);
        orow[c + ch] = to_elem<T>(acc[1][k]);
        orow[2 * c + ch] = to_elem<T>(acc[2][k]);
        orow[3 * c + ch] = xrow[3 * c + ch];               // Eq. 4: identity branch
      }
    }
#pragma unroll
    for (int s = 0; s < NS; ++s) idx[s] = idx_next[s];
    in_grid = in_grid_next;
  }
}

template <typename... KArgs, typename... Args>
cudaError_t launch_chained(void (*kernel)(KArgs...), unsigned blocks, unsigned threads, size_t smem, cudaStream_t st,
                           Args... args) {
  cudaLaunchAttribute pdl[1];
  pdl[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  pdl[0].val.programmaticStreamSerializationAllowed = 1;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(blocks);
  cfg.blockDim = dim3(threads);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cfg.attrs = pdl;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

template <typename T>
cudaError_t cwi_launch(const void* x, const int32_t* coords, int N, int C, Geom g, int S_h, int S_w, const float* w_h,
                       const float* w_w, const float* w_3, void* out, int32_t* grid, cudaStream_t st) {
  const size_t cells = (size_t)g.batch * g.gz * g.gh * g.gw;
  const size_t n16 = (cells * 4 + 15) / 16;
  unsigned fb = (unsigned)((n16 + 1023) / 1024);
  if (fb > 2368) fb = 2368;
  cudaError_t e = launch_chained(sla_cwi_fill_kernel, fb, 256, 0, st, (uint4*)grid, n16);
  if (e != cudaSuccess) return e;
  e = launch_chained(sla_cwi_scatter_kernel, (unsigned)((N + 255) / 256), 256, 0, st, (const int4*)coords, N, g, grid);
  if (e != cudaSuccess) return e;
  const int c = C / 4;
  const size_t smem = (size_t)(S_h + S_w + 29) * c * sizeof(float);
  unsigned blocks = (unsigned)((N + kCwiWarps - 1) / kCwiWarps);
  if (blocks > 592) blocks = 592;                        // 4 x 148 blocks of 16 warps: every warp walks ~6 voxels per 60 000,
                                                         // so the per-block weight staging and per-warp tap set-up are amortised
  const int cpl = (c + 31) / 32;
#define SLA_CWI_LAUNCH(CPL, NS)                                                                                    \
  launch_chained(sla_cwi_conv_kernel<T, CPL, NS>, blocks, 32 * kCwiWarps, smem, st, (const T*)x, (const int4*)coords, \
                 N, C, g, S_h, S_w, w_h, w_w, w_3, (const int32_t*)grid, (T*)out)
#define SLA_CWI_SLOTS(CPL)                     \
  switch (ns) {                                \
    case 1: return SLA_CWI_LAUNCH(CPL, 1);     \
    case 2: return SLA_CWI_LAUNCH(CPL, 2);     \
    case 3: return SLA_CWI_LAUNCH(CPL, 3);     \
    default: return SLA_CWI_LAUNCH(CPL, 4);    \
  }
  const int ns = (S_h + S_w + 29 + 31) / 32;
  switch (cpl) {
    case 1: SLA_CWI_SLOTS(1)
    case 2: SLA_CWI_SLOTS(2)
    case 3: SLA_CWI_SLOTS(3)
    default: SLA_CWI_SLOTS(4)
  }
#undef SLA_CWI_SLOTS
#undef SLA_CWI_LAUNCH
}

}  // namespace

cudaError_t launch_cwi(const void* x, const int32_t* coords, int N, int C, int dt, int batch, int gz, int gh, int gw,
                       int S_h, int S_w, const float* w_h, const float* w_w, const float* w_3, void* out,
                       int32_t* grid, cudaStream_t st) {
  const Geom g{batch, gz, gh, gw};
  if (dt == SLA_F32) return cwi_launch<float>(x, coords, N, C, g, S_h, S_w, w_h, w_w, w_3, out, grid, st);
  if (dt == SLA_F16) return cwi_launch<__half>(x, coords, N, C, g, S_h, S_w, w_h, w_w, w_3, out, grid, st);
  return cwi_launch<__nv_bfloat16>(x, coords, N, C, g, S_h, S_w, w_h, w_w, w_3, out, grid, st);
}

}  // namespace sla
