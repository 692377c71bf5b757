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

__global__ void __launch_bounds__(256) sla_cwi_fill_kernel(uint4* __restrict__ p, size_t n16, unsigned word) {
  pdl_launch_dependents();
  pdl_wait();   // a previous call's conv kernel may still be reading the grid
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n16; i += (size_t)gridDim.x * blockDim.x)
    p[i] = make_uint4(word, word, word, word);
}

struct Geom { int batch, gz, gh, gw; };

__device__ __forceinline__ long long cell_of(const Geom& g, int b, int z, int y, int x) {
  const bool inside = (unsigned)b < (unsigned)g.batch && (unsigned)z < (unsigned)g.gz && (unsigned)y < (unsigned)g.gh &&
                      (unsigned)x < (unsigned)g.gw;
  return inside ? (((long long)b * g.gz + z) * g.gh + y) * g.gw + x : -1;
}

// zmask != nullptr (grid_z <= 32): one word per (b, y, x) column, bit z = "a voxel sits in cell z".  Then only this
// word array is cleared per call (4 bytes per column instead of 4 bytes per cell) and a cell of the index grid is read
// only where its bit is set, so whatever an earlier call or anybody else left in the other cells is never looked at.
__global__ void __launch_bounds__(256)
sla_cwi_scatter_kernel(const int4* __restrict__ coords, int N, Geom g, int32_t* __restrict__ grid,
                       uint32_t* __restrict__ zmask) {
  pdl_launch_dependents();
  pdl_wait();
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  const int4 c = __ldg(coords + i);                      // (b, z, y, x)
  const long long cell = cell_of(g, c.x, c.y, c.z, c.w);
  if (cell >= 0) {                                       // a voxel outside the grid is seen by nobody
    grid[cell] = (int)i;
    if (zmask != nullptr) atomicOr(zmask + ((long long)c.x * g.gh + c.z) * g.gw + c.w, 1u << c.y);
  }
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

// ---- 16-bit rows of 64, 128 or 256 channels: one row per warp-wide load ------------------------------------------------
// Lane l owns V = C / 32 consecutive channels of the row (4, 8 or 16 bytes), which all belong to branch l / 8, so one
// load per lane reads a whole 2C-byte row and the three convolution branches walk their own taps AT THE SAME TIME: in
// step n the eight lanes of branch b fetch the row of the n-th present tap of branch b.  The number of steps is the
// largest tap count of a branch instead of the sum over the branches, and every step moves V channels per lane instead
// of one.  Per (branch, channel) the terms are added in the order of the kernel above (centre, then ascending taps):
// the two kernels give the same bits.
template <typename T> __device__ __forceinline__ float2 unpack2(uint32_t u);
template <> __device__ __forceinline__ float2 unpack2<__half>(uint32_t u) {
  return __half22float2(*reinterpret_cast<const __half2*>(&u));
}
template <> __device__ __forceinline__ float2 unpack2<__nv_bfloat16>(uint32_t u) {
  return make_float2(__uint_as_float(u << 16), __uint_as_float(u & 0xffff0000u));
}
template <typename T> __device__ __forceinline__ uint32_t pack2(float a, float b);
template <> __device__ __forceinline__ uint32_t pack2<__half>(float a, float b) {
  const __half2 h = __floats2half2_rn(a, b);
  return *reinterpret_cast<const uint32_t*>(&h);
}
template <> __device__ __forceinline__ uint32_t pack2<__nv_bfloat16>(float a, float b) {
  const __nv_bfloat162 h = __floats2bfloat162_rn(a, b);
  return *reinterpret_cast<const uint32_t*>(&h);
}
template <int V> __device__ __forceinline__ void ld_row(const void* p, uint32_t (&r)[V / 2]) {
  if constexpr (V == 2) {
    r[0] = __ldg(reinterpret_cast<const uint32_t*>(p));
  } else if constexpr (V == 4) {
    const uint2 t = __ldg(reinterpret_cast<const uint2*>(p));
    r[0] = t.x; r[1] = t.y;
  } else {
    const uint4 t = __ldg(reinterpret_cast<const uint4*>(p));
    r[0] = t.x; r[1] = t.y; r[2] = t.z; r[3] = t.w;
  }
}
template <int V> __device__ __forceinline__ void st_row(void* p, const uint32_t (&r)[V / 2]) {
  if constexpr (V == 2) *reinterpret_cast<uint32_t*>(p) = r[0];
  else if constexpr (V == 4) *reinterpret_cast<uint2*>(p) = make_uint2(r[0], r[1]);
  else *reinterpret_cast<uint4*>(p) = make_uint4(r[0], r[1], r[2], r[3]);
}

// V = C / 32 channels per lane (2, 4, 8).  The taps other than the centres are laid out by POSITION so that every
// branch sits inside one 32-bit ballot: positions 0..25 the 3x3x3 taps, 32.. the S_h taps along y, then the S_w taps
// along x (S_h + S_w <= 32); lane l looks up positions l and 32 + l; the weights are staged in position order.
template <typename T, int V>
__global__ void __launch_bounds__(32 * kCwiWarps, V == 8 ? 1 : 2)
sla_cwi_conv_rows_kernel(const T* __restrict__ x, const int4* __restrict__ coords, int N, Geom g, int S_h, int S_w,
                         const float* __restrict__ w_h, const float* __restrict__ w_w, const float* __restrict__ w_3,
                         const int32_t* __restrict__ grid, const uint32_t* __restrict__ zmask, T* __restrict__ out) {
  extern __shared__ __align__(16) float s_w[];           // [32 + S_h + S_w][c]
  pdl_launch_dependents();
  constexpr int C = 32 * V, c = 8 * V;
  const int Th = S_h + 1, Tw = S_w + 1, P = 32 + S_h + S_w;
  // position -> branch and tap of that branch's kernel (the centre tap is skipped)
  auto tap_of = [&](int p, int& br, int& t) -> bool {
    if (p < 26) { br = 2; t = p + (p >= 13); return true; }
    int q = p - 32;
    if (q < 0) return false;
    if (q < S_h) { br = 0; t = q + (q >= (S_h >> 1)); return true; }
    q -= S_h;
    if (q < S_w) { br = 1; t = q + (q >= (S_w >> 1)); return true; }
    return false;
  };
  for (int i = threadIdx.x; i < P * c; i += blockDim.x) {
    const int p = i / c, ch = i - p * c;
    int br = 0, t = 0;
    float v = 0.f;
    if (tap_of(p, br, t))
      v = br == 0 ? __ldg(w_h + ch * Th + t) : br == 1 ? __ldg(w_w + ch * Tw + t) : __ldg(w_3 + ch * 27 + t);
    s_w[i] = v;
  }
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int br = lane >> 3;                              // branch of this lane's channels (3: identity)
  const int ch0 = (lane & 7) * V;                        // the first of them inside the branch
  const int myslot = br == 2 ? 0 : 1;
  const unsigned mine = br == 2 ? 0x03ffffffu
                      : br == 0 ? (unsigned)((1ull << S_h) - 1ull)
                      : br == 1 ? (unsigned)(((1ull << S_w) - 1ull) << S_h) : 0u;
  float wc[V];                                           // centre weights of this lane's channels
#pragma unroll
  for (int k = 0; k < V; ++k)
    wc[k] = br == 0 ? __ldg(w_h + (ch0 + k) * Th + (S_h >> 1)) : br == 1 ? __ldg(w_w + (ch0 + k) * Tw + (S_w >> 1))
          : br == 2 ? __ldg(w_3 + (ch0 + k) * 27 + 13) : 0.f;
  // per-lane constants of the voxel loop, pinned to registers (ptxas otherwise re-derives them from the thread index
  // and the parameter bank in every iteration and every tap step: a third of the loop's instructions)
  uint32_t wbase = (uint32_t)__cvta_generic_to_shared(s_w + myslot * 32 * c + ch0);
  const T* xl = x + lane * V;
  T* ol = out + lane * V;
  int tdz[2], tdy[2], tdx[2], tdelta[2], tcol[2];
#pragma unroll
  for (int s = 0; s < 2; ++s) {
    int b = 0, t = 0, dz = 1 << 20, dy = 0, dx = 0;        // no tap at this position: always outside the grid
    if (tap_of(lane + 32 * s, b, t)) {
      dz = 0;
      if (b == 0) dy = t - (S_h >> 1);
      else if (b == 1) dx = t - (S_w >> 1);
      else { dz = t / 9 - 1; dy = (t / 3) % 3 - 1; dx = t % 3 - 1; }
    }
    tdz[s] = dz; tdy[s] = dy; tdx[s] = dx;
    tdelta[s] = (dz * g.gh + dy) * g.gw + dx;
    tcol[s] = dy * g.gw + dx;
    asm volatile("" : "+r"(tdelta[s]));
    asm volatile("" : "+r"(tcol[s]));
  }
  asm volatile("" : "+r"(wbase));
  asm volatile("" : "+l"(xl));
  asm volatile("" : "+l"(ol));
  pdl_wait();
  __syncthreads();
  // Look-ups of this lane's two positions around a voxel, in two dependent rounds that belong to different iterations of
  // the voxel loop: round 1 reads the occupancy words of the two columns (0 where the position is outside the grid),
  // round 2 reads the index grid where the position's z bit is set (-1 elsewhere).  < 2^31 cells (host).
  auto columns_of = [&](const int4& me, int& cell0, int& z, unsigned (&m)[2]) {
    const bool me_in = (unsigned)me.x < (unsigned)g.batch && (unsigned)me.y < (unsigned)g.gz &&
                       (unsigned)me.z < (unsigned)g.gh && (unsigned)me.w < (unsigned)g.gw;
    const int col0 = (me.x * g.gh + me.z) * g.gw + me.w;
    cell0 = ((me.x * g.gz + me.y) * g.gh + me.z) * g.gw + me.w;
    z = me_in ? me.y : -1;                                 // -1: the voxel is off the grid
#pragma unroll
    for (int s = 0; s < 2; ++s) {
      const bool inside = me_in && (unsigned)(me.y + tdz[s]) < (unsigned)g.gz &&
                          (unsigned)(me.z + tdy[s]) < (unsigned)g.gh && (unsigned)(me.w + tdx[s]) < (unsigned)g.gw;
      m[s] = inside ? zmask[col0 + tcol[s]] : 0u;
    }
  };
  auto cells_of = [&](int cell0, int z, const unsigned (&m)[2], int (&idx)[2]) {
#pragma unroll
    for (int s = 0; s < 2; ++s)
      idx[s] = ((m[s] >> ((z + tdz[s]) & 31)) & 1u) ? grid[cell0 + tdelta[s]] : -1;
  };
  const int stride = (int)gridDim.x * kCwiWarps;         // N < 2^30 (host): i + 3 stride cannot overflow
  int i = (int)blockIdx.x * kCwiWarps + warp;
  const int4 none = make_int4(-1, -1, -1, -1);           // outside every grid: nothing is loaded for it
  auto coords_of = [&](int j) -> int4 { return j < N ? __ldg(coords + j) : none; };
  // Software pipeline: while voxel i is accumulated, the index-grid cells of voxel i + stride, the occupancy words of
  // voxel i + 2 stride and the coordinates of voxel i + 3 stride are in flight.
  int idx[2], cell1, z1, z0;
  unsigned m1[2];
  {
    unsigned m0[2];
    int cell0;
    columns_of(coords_of(i), cell0, z0, m0);
    cells_of(cell0, z0, m0, idx);
  }
  columns_of(coords_of(i + stride), cell1, z1, m1);
  int4 me2 = coords_of(i + 2 * stride);
  for (; i < N; i += stride) {
    const bool in_grid = z0 >= 0;
    int idx_next[2];
    cells_of(cell1, z1, m1, idx_next);
    z0 = z1;
    columns_of(me2, cell1, z1, m1);
    me2 = coords_of(i + 3 * stride);
    uint32_t own[V / 2];
    ld_row<V>(xl + (size_t)i * C, own);
    float acc[V];
#pragma unroll
    for (int k = 0; k < V / 2; ++k) {                      // centre tap
      const float2 f = unpack2<T>(own[k]);
      acc[2 * k] = wc[2 * k] * f.x;
      acc[2 * k + 1] = wc[2 * k + 1] * f.y;
    }
    const unsigned b0 = __ballot_sync(0xffffffffu, idx[0] >= 0), b1 = __ballot_sync(0xffffffffu, idx[1] >= 0);
    unsigned present = (myslot ? b1 : b0) & mine;          // this branch's taps that hit a voxel
    if (__builtin_expect(!in_grid, 0)) {                   // a voxel off the grid: zeros (it has no neighbour either)
#pragma unroll
      for (int k = 0; k < V; ++k) acc[k] = 0.f;
    }
    const int steps = __reduce_max_sync(0xffffffffu, __popc(present));
    // Ascending taps per branch (deterministic sums), four steps at a time: the rows of all four are requested before
    // the first is used (the loop is bound by the latency of these L2 reads, not by instruction issue).
    for (int n = 0; n < steps; n += 4) {
      uint32_t r[4][V / 2];
      int lt[4];
      bool lv[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        lv[u] = false;
        lt[u] = 0;
        if (u == 0 || n + u < steps) {                     // warp-uniform
          lv[u] = present != 0;
          lt[u] = __ffs(present) - 1;                      // -1 (list ended): the shuffles read lane 31, unused
          present &= present - 1;
          const int j0 = __shfl_sync(0xffffffffu, idx[0], lt[u]), j1 = __shfl_sync(0xffffffffu, idx[1], lt[u]);
          if (lv[u]) ld_row<V>(xl + (size_t)(myslot ? j1 : j0) * C, r[u]);
        }
      }
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        if (lv[u]) {
          float wt[V];
          const uint32_t wa = wbase + (uint32_t)lt[u] * (c * 4u);
          if constexpr (V == 2) {
            asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(wt[0]), "=f"(wt[1]) : "r"(wa));
          } else {
#pragma unroll
            for (int k = 0; k < V; k += 4)
              asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];"
                           : "=f"(wt[k]), "=f"(wt[k + 1]), "=f"(wt[k + 2]), "=f"(wt[k + 3]) : "r"(wa + 4u * k));
          }
#pragma unroll
          for (int k = 0; k < V / 2; ++k) {
            const float2 f = unpack2<T>(r[u][k]);
            acc[2 * k] = fmaf(wt[2 * k], f.x, acc[2 * k]);
            acc[2 * k + 1] = fmaf(wt[2 * k + 1], f.y, acc[2 * k + 1]);
          }
        }
      }
    }
    if (br < 3) {                                          // Eq. 4: the identity branch keeps the input's bits
#pragma unroll
      for (int k = 0; k < V / 2; ++k) own[k] = pack2<T>(acc[2 * k], acc[2 * k + 1]);
    }
    st_row<V>(ol + (size_t)i * C, own);
    idx[0] = idx_next[0]; idx[1] = idx_next[1];
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

// The convolution kernels are persistent: as many blocks as the device holds at once (register-bound: 2 per SM for
// most instantiations), so the weights are staged once per resident block and no block waits for a second wave.
template <typename... KArgs, typename... Args>
cudaError_t launch_conv(void (*kernel)(KArgs...), int N, size_t smem, cudaStream_t st, Args... args) {
  int dev = 0, sms = 148, per_sm = 1;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
    sms = 148;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, 32 * kCwiWarps, smem) != cudaSuccess || per_sm < 1)
    per_sm = 1;
  unsigned blocks = (unsigned)((N + kCwiWarps - 1) / kCwiWarps);
  if (blocks > (unsigned)(sms * per_sm)) blocks = (unsigned)(sms * per_sm);
  return launch_chained(kernel, blocks, 32 * kCwiWarps, smem, st, args...);
}

template <typename T>
cudaError_t cwi_launch(const void* x, const int32_t* coords, int N, int C, Geom g, int S_h, int S_w, const float* w_h,
                       const float* w_w, const float* w_3, void* out, int32_t* grid, uint32_t* zmask, cudaStream_t st) {
  const size_t cells = (size_t)g.batch * g.gz * g.gh * g.gw;
  const int c = C / 4;
  const size_t smem = (size_t)(S_h + S_w + 29) * c * sizeof(float);
  const int cpl = (c + 31) / 32;
  const int ns = (S_h + S_w + 29 + 31) / 32;
  auto fill = [&](void* p, size_t bytes, unsigned word) -> cudaError_t {
    const size_t n16 = (bytes + 15) / 16;
    unsigned fb = (unsigned)((n16 + 1023) / 1024);
    if (fb > 2368) fb = 2368;
    if (fb == 0) fb = 1;
    return launch_chained(sla_cwi_fill_kernel, fb, 256, 0, st, (uint4*)p, n16, word);
  };
  const unsigned sblocks = (unsigned)((N + 255) / 256);
  if constexpr (sizeof(T) == 2) {
    const bool aligned = (((uintptr_t)x | (uintptr_t)out) & 15) == 0;
    if (S_h + S_w <= 32 && g.gz <= 32 && cells < (1ull << 31) && N < (1 << 30) && aligned &&
        (C == 64 || C == 128 || C == 256)) {
      // a row is one 4-, 8- or 16-byte load per lane; occupancy words instead of a cleared index grid
      cudaError_t e = fill(zmask, (size_t)g.batch * g.gh * g.gw * 4, 0u);
      if (e != cudaSuccess) return e;
      e = launch_chained(sla_cwi_scatter_kernel, sblocks, 256, 0, st, (const int4*)coords, N, g, grid, zmask);
      if (e != cudaSuccess) return e;
      const size_t smem_rows = (size_t)(32 + S_h + S_w) * c * sizeof(float);
#define SLA_CWI_ROWS(V)                                                                                    \
  launch_conv(sla_cwi_conv_rows_kernel<T, V>, N, smem_rows, st, (const T*)x, (const int4*)coords, N, g, S_h, S_w, w_h, \
              w_w, w_3, (const int32_t*)grid, (const uint32_t*)zmask, (T*)out)
      if (C == 64) return SLA_CWI_ROWS(2);
      if (C == 128) return SLA_CWI_ROWS(4);
      return SLA_CWI_ROWS(8);
#undef SLA_CWI_ROWS
    }
  }
  cudaError_t e = fill(grid, cells * 4, 0xFFFFFFFFu);
  if (e != cudaSuccess) return e;
  e = launch_chained(sla_cwi_scatter_kernel, sblocks, 256, 0, st, (const int4*)coords, N, g, grid, (uint32_t*)nullptr);
  if (e != cudaSuccess) return e;
#define SLA_CWI_LAUNCH(CPL, NS)                                                                                    \
  launch_conv(sla_cwi_conv_kernel<T, CPL, NS>, N, smem, st, (const T*)x, (const int4*)coords, \
                 N, C, g, S_h, S_w, w_h, w_w, w_3, (const int32_t*)grid, (T*)out)
#define SLA_CWI_SLOTS(CPL)                     \
  switch (ns) {                                \
    case 1: return SLA_CWI_LAUNCH(CPL, 1);     \
    case 2: return SLA_CWI_LAUNCH(CPL, 2);     \
    case 3: return SLA_CWI_LAUNCH(CPL, 3);     \
    default: return SLA_CWI_LAUNCH(CPL, 4);    \
  }
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
                       int32_t* grid, uint32_t* zmask, cudaStream_t st) {
  const Geom g{batch, gz, gh, gw};
  if (dt == SLA_F32) return cwi_launch<float>(x, coords, N, C, g, S_h, S_w, w_h, w_w, w_3, out, grid, zmask, st);
  if (dt == SLA_F16) return cwi_launch<__half>(x, coords, N, C, g, S_h, S_w, w_h, w_w, w_3, out, grid, zmask, st);
  return cwi_launch<__nv_bfloat16>(x, coords, N, C, g, S_h, S_w, w_h, w_w, w_3, out, grid, zmask, st);
}

}  // namespace sla
