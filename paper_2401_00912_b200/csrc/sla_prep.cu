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
sla_offsets_kernel(const int32_t* __restrict__ win_id, int N, int W, int32_t* __restrict__ off) {
  // Programmatic dependent launch: a following kernel that opted in (sla_fwd_tc_kernel) may become
  // resident now; it still waits for this whole grid (griddepcontrol.wait) before it reads `off`.
  asm volatile("griddepcontrol.launch_dependents;");
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i > N) return;
  const int lo = (i == 0) ? 0 : __ldg(win_id + i - 1) + 1;
  const int hi = (i == N) ? W : __ldg(win_id + i);
  for (int w = lo; w <= hi; ++w) off[w] = i;
}

}  // namespace

cudaError_t launch_offsets(const int32_t* win_id, int N, int W, int32_t* off, cudaStream_t st) {
  const int threads = 256;
  const int blocks = (N + 1 + threads - 1) / threads;
  sla_offsets_kernel<<<blocks, threads, 0, st>>>(win_id, N, W, off);
  return cudaGetLastError();
}

}  // namespace sla
