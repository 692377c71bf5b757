// sla_prep.cu -- "offsets generation" (Fig. 5): window id of every voxel -> window
// offsets of the flat window-sorted sequence.  Integer only, bit-exact.
//
//   off[w] = #{ i : win_id[i] < w },  w = 0..W      (win_id non-decreasing, each in [0,W))
//
// One coalesced pass over the ids: position i (0..N) is a boundary between id[i-1] and id[i] (with
// id[-1] = -1 and id[N] = W); every w in (id[i-1], id[i]] has exactly i ids below it, so the thread
// at i writes off[w] = i for those w (more than one only where ids skip, i.e. empty windows).
#include "sla_internal.cuh"

namespace sla {
namespace {

__global__ void __launch_bounds__(256)
sla_offsets_kernel(const int32_t* __restrict__ win_id, int N, int W, int32_t* __restrict__ off, int id_base) {
  // Programmatic dependent launch: a following kernel that opted in (sla_fwd_tc_kernel) may become
  // resident now; it still waits for this whole grid (griddepcontrol.wait) before it reads `off`.
  asm volatile("griddepcontrol.launch_dependents;");
  const long long i64 = (long long)blockIdx.x * blockDim.x + threadIdx.x;   // N may be within 256 of 2^31
  if (i64 > N) return;
  const int i = (int)i64;
  // ids outside [0, W) violate the precondition; clamp so that they can never write out of bounds
  // id_base: the ids are window indices of a longer scene; this call covers windows id_base .. id_base+W-1 of it
  const int lo = (i == 0) ? 0 : max(0, min(W, __ldg(win_id + i - 1) - id_base) + 1);
  const int hi = (i == N) ? W : max(-1, min(W, __ldg(win_id + i) - id_base));
  for (int w = lo; w <= hi; ++w) off[w] = i;
}

// Size-matched streaming ceiling: reads three tensors and writes one -- the forward's
// 3:1 traffic mix -- with 128-bit accesses and nothing else: out = a ^ b ^ c.  Every thread issues its 12
// loads before the first use, so a block has 6 KB per tensor in flight; no shared memory, so several
// blocks are resident per SM.  What this kernel cannot reach on a problem of the same size under the same
// timing protocol, no SLA kernel can.
constexpr int kCeilThreads = 512, kCeilUnroll = 4;
__global__ void __launch_bounds__(kCeilThreads)
sla_stream_ceiling_kernel(const uint4* __restrict__ a, const uint4* __restrict__ b, const uint4* __restrict__ c,
                          uint4* __restrict__ out, size_t n16) {
  const size_t base = (size_t)blockIdx.x * (kCeilThreads * kCeilUnroll) + threadIdx.x;
  uint4 x[kCeilUnroll], y[kCeilUnroll], z[kCeilUnroll];
#pragma unroll
  for (int u = 0; u < kCeilUnroll; ++u) {
    const size_t i = base + (size_t)u * kCeilThreads;
    if (i < n16) {
      asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                   : "=r"(x[u].x), "=r"(x[u].y), "=r"(x[u].z), "=r"(x[u].w) : "l"(a + i));
      asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                   : "=r"(y[u].x), "=r"(y[u].y), "=r"(y[u].z), "=r"(y[u].w) : "l"(b + i));
      asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                   : "=r"(z[u].x), "=r"(z[u].y), "=r"(z[u].z), "=r"(z[u].w) : "l"(c + i));
    }
  }
#pragma unroll
  for (int u = 0; u < kCeilUnroll; ++u) {
    const size_t i = base + (size_t)u * kCeilThreads;
    if (i < n16)
      out[i] = make_uint4(x[u].x ^ y[u].x ^ z[u].x, x[u].y ^ y[u].y ^ z[u].y, x[u].z ^ y[u].z ^ z[u].z,
                          x[u].w ^ y[u].w ^ z[u].w);
  }
}

// Zero the fp32 state slots of the workspace.  A kernel rather than a memset node so that it can sit in the chain of
// programmatic dependent launches: the forward/backward kernel behind it becomes resident and sets itself up while
// this one runs, and this one does the same behind whatever precedes it in the stream.
__global__ void __launch_bounds__(256) sla_zero_kernel(uint4* __restrict__ p, size_t n16) {
  asm volatile("griddepcontrol.launch_dependents;");
  asm volatile("griddepcontrol.wait;" ::: "memory");   // a previous call's kernels may still be reading the workspace
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n16; i += (size_t)gridDim.x * blockDim.x)
    p[i] = make_uint4(0u, 0u, 0u, 0u);
}

}  // namespace

cudaError_t launch_zero(void* p, size_t bytes, cudaStream_t st) {
  const size_t n16 = (bytes + 15) / 16;                    // the workspace size is a multiple of 16
  if (n16 == 0) return cudaSuccess;
  unsigned blocks = (unsigned)((n16 + 1023) / 1024);
  if (blocks > 592) blocks = 592;
  cudaLaunchAttribute pdl[1];
  pdl[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  pdl[0].val.programmaticStreamSerializationAllowed = 1;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(blocks);
  cfg.blockDim = dim3(256);
  cfg.stream = st;
  cfg.attrs = pdl;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, sla_zero_kernel, (uint4*)p, n16);
}

cudaError_t launch_stream_ceiling(const void* a, const void* b, const void* c, void* out, size_t bytes,
                                  cudaStream_t st) {
  const size_t n16 = bytes / 16;
  const size_t per_block = (size_t)kCeilThreads * kCeilUnroll;
  const unsigned blocks = (unsigned)((n16 + per_block - 1) / per_block);
  if (blocks == 0) return cudaSuccess;
  sla_stream_ceiling_kernel<<<blocks, kCeilThreads, 0, st>>>((const uint4*)a, (const uint4*)b, (const uint4*)c,
                                                            (uint4*)out, n16);
  return cudaGetLastError();
}

cudaError_t launch_offsets(const int32_t* win_id, int N, int W, int32_t* off, cudaStream_t st, int id_base) {
  const int threads = 256;
  const unsigned blocks = (unsigned)(((long long)N + 1 + threads - 1) / threads);
  sla_offsets_kernel<<<blocks, threads, 0, st>>>(win_id, N, W, off, id_base);
  return cudaGetLastError();
}

}  // namespace sla
