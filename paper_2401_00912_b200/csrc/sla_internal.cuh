// sla_internal.cuh -- shared device helpers of the CUDA path (dtype traits, feature map, launch
// declarations).  Product code: shares nothing with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <cuda_fp16.h>
#include <cuda_bf16.h>
#include <stdint.h>

#include "../../include/sla.h"

namespace sla {

// ---- dtype traits: load/store one element as fp32 ------------------------------------------------
template <typename T> struct Elem;
template <> struct Elem<float> {
  static __device__ __forceinline__ float ld(const float* p) { return __ldg(p); }
  static __device__ __forceinline__ void st(float* p, float x) { *p = x; }
};
template <> struct Elem<__half> {
  static __device__ __forceinline__ float ld(const __half* p) {
    return __half2float(__ushort_as_half(__ldg(reinterpret_cast<const unsigned short*>(p))));
  }
  static __device__ __forceinline__ void st(__half* p, float x) { *p = __float2half_rn(x); }
};
template <> struct Elem<__nv_bfloat16> {
  static __device__ __forceinline__ float ld(const __nv_bfloat16* p) {
    return __uint_as_float(((unsigned)__ldg(reinterpret_cast<const unsigned short*>(p))) << 16);
  }
  static __device__ __forceinline__ void st(__nv_bfloat16* p, float x) { *p = __float2bfloat16_rn(x); }
};

// ---- feature map phi(x) = elu(x)+1 (reading A1; Eq. 3 cites [17]) and its derivative --
// fp32 path: full-precision expf (the fp32 tolerance is 1e-5 relative).
// `relu` selects the second map ("Efficient Attn [3]"): phi(x) = max(x, 0).
__device__ __forceinline__ float phi_f32(float x, bool relu) {
  return relu ? fmaxf(x, 0.f) : (x > 0.f ? x + 1.f : expf(x));
}
__device__ __forceinline__ float dphi_f32(float x, bool relu) {
  return relu ? (x > 0.f ? 1.f : 0.f) : (x > 0.f ? 1.f : expf(x));
}

// ---- window search: largest w in [0,W) with off[w] <= row  (off[0]=0 <= row < off[W]) -------------
__device__ __forceinline__ int window_of_row(const int32_t* __restrict__ off, int W, int row) {
  int lo = 0, hi = W;  // invariant: off[lo] <= row < off[hi]
  while (hi - lo > 1) {
    int mid = (lo + hi) >> 1;
    if (__ldg(off + mid) <= row) lo = mid; else hi = mid;
  }
  return lo;
}

// Tiling constants of the generic (CUDA-core, fp32-math) path.
//   TILE_ROWS: rows of the flat sequence per thread block ("chunk", Fig. 3a).
//   FUSE_MAX : a window of at most this many rows is processed whole by the block that owns its
//              first row (state never leaves the SM); longer windows are split by tile and their
//              partial states are reduced in global memory (workspace) with fp32 atomics.
constexpr int kTileRows = 64;
#ifndef SLA_BWD_TILE
#define SLA_BWD_TILE 64
#endif
constexpr int kBwdTileRows = SLA_BWD_TILE;   // backward: rows per thread block
constexpr int kFuseMax = 256;
constexpr int kRowBatch = 8;  // rows staged per inner step
// The workspace starts with a 16-byte header (int flag: 1 = some window was split in this call),
// followed by the fp32 state slots.  Zeroed by the memset at the start of every call.
constexpr int kWsHeaderFloats = 4;

struct Problem {
  const void* q; const void* k; const void* v; const void* g;
  void* out; void* dq; void* dk; void* dv;
  const int32_t* off;
  float* ws_state;   // [W,H,d+1,d] fp32 (S rows 0..d-1, z in row d) for split windows
  float* ws_dstate;  // [W,H,d+1,d] fp32 (dS, dz) for split windows (backward)
  int N, W, H, d;
  int phi;           // sla_feature_map_t
  float eps;         // added to the denominator (0 for SLA_PHI_ELU1)
  bool bounded;      // caller guarantees every window has <= kFuseMax rows: no workspace, no split pass
  const void* span_table;   // optional span table of this scene (sla_build_span_table); nullptr: search in the kernel
  bool tcgen05;      // main pass on the tcgen05 kernel (sla_fwd_umma.cu) instead of the mma.sync kernel
};

// Launchers (defined in the .cu files); all enqueue on `st` and return the last CUDA error.
// zero `bytes` bytes (16-byte aligned) with a kernel that takes part in programmatic dependent launch
cudaError_t launch_zero(void* p, size_t bytes, cudaStream_t st);
cudaError_t launch_offsets(const int32_t* win_id, int N, int W, int32_t* off, cudaStream_t st, int id_base = 0);
cudaError_t launch_forward_generic(const Problem& p, int dt, cudaStream_t st);
cudaError_t launch_backward_generic(const Problem& p, int dt, cudaStream_t st);
bool backward_tc_supported(const Problem& p, int dt);
cudaError_t launch_backward_tc(const Problem& p, int dt, cudaStream_t st);
cudaError_t launch_backward_tc32(const Problem& p, int dt, cudaStream_t st);   // d_h = 32 (sla_bwd_tc32.cu)
bool forward_tc_supported(const Problem& p, int dt);
cudaError_t launch_forward_tc(const Problem& p, int dt, cudaStream_t st);
// span table of the tensor-core forward (SURVEY a1's work list): bytes for a scene, and the kernel that fills it
size_t span_table_bytes(long long N, int H, int d);
cudaError_t launch_span_table(const int32_t* off, int N, int W, int H, int d, void* table, cudaStream_t st);
// tcgen05 main pass of the forward (sla_fwd_umma.cu): fused windows + partial states of long windows
bool forward_umma_supported(const Problem& p, int dt);
cudaError_t launch_forward_umma_main(const Problem& p, int dt, cudaStream_t st);
// measurement aid (sla_bench_stream_ceiling): out = a ^ b ^ c over `bytes` bytes per tensor, 128-bit accesses
// sequence preparation (sla_seq.cu)
size_t sort_workspace_bytes(long long N);
cudaError_t launch_window_keys(const int32_t* coords, int N, int batch, int grid_h, int grid_w, int S_h, int S_w,
                               int32_t* key, cudaStream_t st);
bool sequence_onepass_fits(long long N, long long W, size_t scratch);
cudaError_t launch_sequence_onepass(const int32_t* coords, int N, int batch, int grid_h, int grid_w, int S_h, int S_w,
                                    int32_t* key, void* cnt, int32_t* perm, int32_t* key_sorted, int32_t* off,
                                    cudaStream_t st);
cudaError_t launch_sort_by_key(const int32_t* key, int N, int W, int32_t* perm, int32_t* key_sorted, void* ws,
                               cudaStream_t st);
cudaError_t launch_permute_rows(const void* src, const int32_t* perm, long long N, size_t row_bytes, void* dst,
                                bool scatter, cudaStream_t st);
// shared Q/K/V projection (sla_proj.cu): y = x w^T (+ bias) on tcgen05, split into q, k, v
bool qkv_projection_supported(int C, int dt);
// n_out = 3: w [3C, C] -> q, k, v; n_out = 1: w [C, C] -> q only (a plain linear layer, e.g. the output projection)
cudaError_t launch_qkv_projection(const void* x, const void* w, const float* bias, int N, int C, int dt, int n_out,
                                  void* q, void* k, void* v, cudaStream_t st);
// Cross-Window Interaction (sla_cwi.cu): depth-wise sparse convolutions on the active voxels
cudaError_t launch_cwi(const void* x, const int32_t* coords, int N, int C, int dt, int batch, int gz, int gh, int gw,
                       int S_h, int S_w, const float* w_h, const float* w_w, const float* w_3, void* out,
                       int32_t* grid, uint32_t* zmask, cudaStream_t st);
cudaError_t launch_stream_ceiling(const void* a, const void* b, const void* c, void* out, size_t bytes,
                                  cudaStream_t st);

}  // namespace sla
