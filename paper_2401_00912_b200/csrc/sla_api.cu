// sla_api.cu -- the extern "C" boundary declared in include/sla.h: argument validation, workspace
// carving and kernel dispatch.  No torch types; plain pointers and sizes.
#include <cstdint>
#include <mutex>

#include "sla_internal.cuh"

namespace {

inline size_t esize(int dt) { return dt == SLA_F32 ? 4 : 2; }
inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

// fp32 accumulators for windows split across thread blocks: one slot per possible split window.
inline size_t state_slots(int64_t N) { return (size_t)(N / (sla::kFuseMax + 1)) + 1; }
inline size_t state_bytes(int64_t N, int H, int d) {
  return sla::kWsHeaderFloats * sizeof(float) +
         state_slots(N) * (size_t)H * (size_t)(d + 1) * (size_t)d * sizeof(float);
}

int check_common(int64_t N, int32_t W, int32_t H, int32_t d_h, int dt) {
  if (N < 0 || W < 0 || H < 1 || N >= (int64_t(1) << 31)) return SLA_ERR_INVALID_ARG;
  if (dt != SLA_F32 && dt != SLA_F16 && dt != SLA_BF16) return SLA_ERR_UNSUPPORTED;
  if (d_h != 16 && d_h != 32) return SLA_ERR_UNSUPPORTED;
  if (((size_t)H * d_h * esize(dt)) % 16 != 0) return SLA_ERR_UNSUPPORTED;
  return SLA_OK;
}

// ---- sla_forward_static: the forward's workspace in a file-scope device array, so the call allocates nothing ----
// One array per GPU that loads the library, held until exit.  Every sla_forward_static call on a device shares it.
static __device__ __align__(256) unsigned char g_static_workspace[SLA_STATIC_WORKSPACE_BYTES];

// In host code `g_static_workspace` is only a handle for the symbol, not a device address: the address a kernel may
// use comes from cudaGetSymbolAddress, asked once per device with that device current, here in the array's own file.
int static_workspace(void** ptr) {
  static std::mutex mu;
  static void* addr[64] = {};
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) return SLA_ERR_CUDA;
  if (dev < 0 || dev >= 64) return SLA_ERR_UNSUPPORTED;
  std::lock_guard<std::mutex> lock(mu);
  if (!addr[dev]) {
    void* p = nullptr;
    if (cudaGetSymbolAddress(&p, g_static_workspace) != cudaSuccess || !p) return SLA_ERR_CUDA;
    addr[dev] = p;
  }
  *ptr = addr[dev];
  return SLA_OK;
}

}  // namespace

extern "C" {

const char* sla_status_string(int status) {
  switch (status) {
    case SLA_OK: return "SLA_OK";
    case SLA_ERR_INVALID_ARG: return "SLA_ERR_INVALID_ARG";
    case SLA_ERR_UNSUPPORTED: return "SLA_ERR_UNSUPPORTED";
    case SLA_ERR_WORKSPACE: return "SLA_ERR_WORKSPACE";
    case SLA_ERR_CUDA: return "SLA_ERR_CUDA";
    case SLA_ERR_TOO_LARGE: return "SLA_ERR_TOO_LARGE";
    default: return "SLA_ERR_UNKNOWN";
  }
}

const char* sla_version(void) { return "sla-b200 0.1 (sm_100a)"; }

size_t sla_workspace_bytes(int64_t N, int32_t W, int32_t H, int32_t d_h, int dt, int for_backward) {
  if (check_common(N, W, H, d_h, dt) != SLA_OK) return 0;
  const size_t one = state_bytes(N, H, d_h);
  return for_backward ? 2 * one : one;
}

int sla_offsets_from_window_ids(const int32_t* win_id, int64_t N, int32_t W, int32_t* window_offsets,
                                sla_stream_t stream) {
  if (N < 0 || W < 0 || N >= (int64_t(1) << 31)) return SLA_ERR_INVALID_ARG;
  if (!window_offsets || (N > 0 && !win_id)) return SLA_ERR_INVALID_ARG;
  if (N > 0 && W == 0) return SLA_ERR_INVALID_ARG;
  cudaError_t e = sla::launch_offsets(win_id, (int)N, W, window_offsets, (cudaStream_t)stream);
  return e == cudaSuccess ? SLA_OK : SLA_ERR_CUDA;
}

// ---- sequence preparation ----
static int64_t count_windows(int32_t batch, int32_t grid_h, int32_t grid_w, int32_t S_h, int32_t S_w) {
  if (batch < 1 || grid_h < 1 || grid_w < 1 || S_h < 1 || S_w < 1) return -1;
  const int64_t nwy = ((int64_t)grid_h + S_h - 1) / S_h, nwx = ((int64_t)grid_w + S_w - 1) / S_w;
  const int64_t W = (int64_t)batch * nwy * nwx;
  return W < (int64_t(1) << 31) - 1 ? W : -1;
}

int64_t sla_window_count(int32_t batch, int32_t grid_h, int32_t grid_w, int32_t S_h, int32_t S_w) {
  return count_windows(batch, grid_h, grid_w, S_h, S_w);
}

int sla_window_keys(const int32_t* coords, int64_t N, int32_t batch, int32_t grid_h, int32_t grid_w, int32_t S_h,
                    int32_t S_w, int32_t* key, sla_stream_t stream) {
  if (N < 0 || N >= (int64_t(1) << 31) || count_windows(batch, grid_h, grid_w, S_h, S_w) < 0) return SLA_ERR_INVALID_ARG;
  if (N == 0) return SLA_OK;
  if (!coords || !key) return SLA_ERR_INVALID_ARG;
  if (!aligned16(coords)) return SLA_ERR_UNSUPPORTED;
  cudaError_t e = sla::launch_window_keys(coords, (int)N, batch, grid_h, grid_w, S_h, S_w, key, (cudaStream_t)stream);
  return e == cudaSuccess ? SLA_OK : SLA_ERR_CUDA;
}

size_t sla_sort_workspace_bytes(int64_t N) {
  if (N < 0 || N >= (int64_t(1) << 31)) return 0;
  return sla::sort_workspace_bytes(N);
}

int sla_sort_by_window(const int32_t* key, int64_t N, int32_t W, int32_t* perm, int32_t* key_sorted,
                       void* workspace, size_t workspace_bytes, sla_stream_t stream) {
  if (N < 0 || N >= (int64_t(1) << 31) || W < 0 || W == INT32_MAX) return SLA_ERR_INVALID_ARG;
  if (N == 0) return SLA_OK;
  if (!key || !perm || !key_sorted || key == key_sorted) return SLA_ERR_INVALID_ARG;
  if (!workspace || workspace_bytes < sla::sort_workspace_bytes(N) || !aligned16(workspace)) return SLA_ERR_WORKSPACE;
  cudaError_t e = sla::launch_sort_by_key(key, (int)N, W, perm, key_sorted, workspace, (cudaStream_t)stream);
  return e == cudaSuccess ? SLA_OK : SLA_ERR_CUDA;
}

static int permute_rows(const void* src, const int32_t* perm, int64_t N, size_t row_bytes, void* dst, bool scatter,
                        sla_stream_t stream) {
  if (N < 0 || N >= (int64_t(1) << 31)) return SLA_ERR_INVALID_ARG;
  if (N == 0 || row_bytes == 0) return SLA_OK;
  if (!src || !perm || !dst || src == dst) return SLA_ERR_INVALID_ARG;
  if (row_bytes % 4 != 0 || ((reinterpret_cast<uintptr_t>(src) | reinterpret_cast<uintptr_t>(dst)) & 3u) != 0 ||
      row_bytes / 4 > (size_t)INT32_MAX)
    return SLA_ERR_UNSUPPORTED;
  cudaError_t e = sla::launch_permute_rows(src, perm, N, row_bytes, dst, scatter, (cudaStream_t)stream);
  return e == cudaSuccess ? SLA_OK : SLA_ERR_CUDA;
}

int sla_gather_rows(const void* src, const int32_t* perm, int64_t N, size_t row_bytes, void* dst, sla_stream_t stream) {
  return permute_rows(src, perm, N, row_bytes, dst, false, stream);
}

int sla_scatter_rows(const void* src, const int32_t* perm, int64_t N, size_t row_bytes, void* dst, sla_stream_t stream) {
  return permute_rows(src, perm, N, row_bytes, dst, true, stream);
}

int sla_sequence_from_coords(const int32_t* coords, int64_t N, int32_t batch, int32_t grid_h, int32_t grid_w,
                             int32_t S_h, int32_t S_w, int32_t* perm, int32_t* key_sorted, int32_t* window_offsets,
                             void* workspace, size_t workspace_bytes, sla_stream_t stream) {
  const int64_t W = count_windows(batch, grid_h, grid_w, S_h, S_w);
  if (N < 0 || N >= (int64_t(1) << 31) || W < 0) return SLA_ERR_INVALID_ARG;
  if (!window_offsets || (N > 0 && (!coords || !perm || !key_sorted))) return SLA_ERR_INVALID_ARG;
  if (N > 0 && !aligned16(coords)) return SLA_ERR_UNSUPPORTED;
  const size_t key_bytes = ((size_t)N * 4 + 15) / 16 * 16;
  if (N > 0 && (!workspace || workspace_bytes < key_bytes + sla::sort_workspace_bytes(N) || !aligned16(workspace)))
    return SLA_ERR_WORKSPACE;
  cudaStream_t st = (cudaStream_t)stream;
  int32_t* key = static_cast<int32_t*>(workspace);
  if (sla::sequence_onepass_fits(N, W, N > 0 ? sla::sort_workspace_bytes(N) : 0)) {
    // one scene (W + 1 <= 2048 bins, >= ~1000 voxels so that the counts fit the radix sort's scratch): counting sort in
    // one pass, offsets out of its scan
    cudaError_t e1 = sla::launch_sequence_onepass(coords, (int)N, batch, grid_h, grid_w, S_h, S_w, key,
                                                  static_cast<char*>(workspace) + key_bytes, perm, key_sorted,
                                                  window_offsets, st);
    return e1 == cudaSuccess ? SLA_OK : SLA_ERR_CUDA;
  }
  if (N > 0) {
    if (sla::launch_window_keys(coords, (int)N, batch, grid_h, grid_w, S_h, S_w, key, st) != cudaSuccess) return SLA_ERR_CUDA;
    if (sla::launch_sort_by_key(key, (int)N, (int)W, perm, key_sorted, static_cast<char*>(workspace) + key_bytes, st) != cudaSuccess)
      return SLA_ERR_CUDA;
  }
  // keys equal to W (voxels outside the grid) sort behind every window: off[W] = number of voxels inside
  cudaError_t e = sla::launch_offsets(key_sorted, (int)N, (int)W, window_offsets, st);
  return e == cudaSuccess ? SLA_OK : SLA_ERR_CUDA;
}

size_t sla_sequence_workspace_bytes(int64_t N) {
  if (N < 0 || N >= (int64_t(1) << 31)) return 0;
  return ((size_t)N * 4 + 15) / 16 * 16 + sla::sort_workspace_bytes(N);
}

// ---- shared Q/K/V projection ----
int sla_qkv_projection(const void* x, const void* w_qkv, const float* bias, int64_t N, int32_t C, int dt, void* q,
                       void* k, void* v, sla_stream_t stream) {
  if (N < 0 || N >= (int64_t(1) << 31) || C < 1) return SLA_ERR_INVALID_ARG;
  if (!sla::qkv_projection_supported(C, dt)) return SLA_ERR_UNSUPPORTED;
  if (N == 0) return SLA_OK;
  if (!x || !w_qkv || !q || !k || !v) return SLA_ERR_INVALID_ARG;
  if (!aligned16(x) || !aligned16(w_qkv) || !aligned16(q) || !aligned16(k) || !aligned16(v) || !aligned16(bias))
    return SLA_ERR_UNSUPPORTED;
  cudaError_t e = sla::launch_qkv_projection(x, w_qkv, bias, (int)N, C, dt, 3, q, k, v, (cudaStream_t)stream);
  return e == cudaSuccess ? SLA_OK : SLA_ERR_CUDA;
}

int sla_linear(const void* x, const void* w, const float* bias, int64_t N, int32_t C, int dt, void* y,
               sla_stream_t stream) {
  if (N < 0 || N >= (int64_t(1) << 31) || C < 1) return SLA_ERR_INVALID_ARG;
  if (!sla::qkv_projection_supported(C, dt)) return SLA_ERR_UNSUPPORTED;
  if (N == 0) return SLA_OK;
  if (!x || !w || !y || x == y) return SLA_ERR_INVALID_ARG;
  if (!aligned16(x) || !aligned16(w) || !aligned16(y) || !aligned16(bias)) return SLA_ERR_UNSUPPORTED;
  cudaError_t e = sla::launch_qkv_projection(x, w, bias, (int)N, C, dt, 1, y, nullptr, nullptr, (cudaStream_t)stream);
  return e == cudaSuccess ? SLA_OK : SLA_ERR_CUDA;
}

// ---- Cross-Window Interaction ----
static int64_t cwi_cells(int32_t batch, int32_t gz, int32_t gh, int32_t gw) {
  if (batch < 1 || gz < 1 || gh < 1 || gw < 1) return -1;
  const int64_t a = (int64_t)batch * gz, b = (int64_t)gh * gw;
  if (a > (int64_t(1) << 31) / b) return -1;
  return a * b < (int64_t(1) << 31) ? a * b : -1;
}

size_t sla_cwi_workspace_bytes(int32_t batch, int32_t grid_z, int32_t grid_h, int32_t grid_w) {
  const int64_t cells = cwi_cells(batch, grid_z, grid_h, grid_w);
  if (cells < 0) return 0;
  // the index grid (4 bytes per cell) + one occupancy word per (b, y, x) column
  return ((size_t)cells * 4 + 15) / 16 * 16 + ((size_t)batch * grid_h * grid_w * 4 + 15) / 16 * 16;
}

int sla_cwi_forward(const void* x, const int32_t* coords, int64_t N, int32_t C, int dt, int32_t batch, int32_t grid_z,
                    int32_t grid_h, int32_t grid_w, int32_t S_h, int32_t S_w, const float* w_h, const float* w_w,
                    const float* w_3, void* out, void* workspace, size_t workspace_bytes, sla_stream_t stream) {
  if (N < 0 || N >= (int64_t(1) << 31) || C < 4 || cwi_cells(batch, grid_z, grid_h, grid_w) < 0)
    return SLA_ERR_INVALID_ARG;
  if (S_h < 0 || S_w < 0 || (S_h & 1) || (S_w & 1)) return SLA_ERR_INVALID_ARG;   // even windows: odd, centred kernels
  if (dt != SLA_F32 && dt != SLA_F16 && dt != SLA_BF16) return SLA_ERR_UNSUPPORTED;
  if (C % 4 != 0 || C > 512 || S_h + S_w + 29 > 128) return SLA_ERR_UNSUPPORTED;
  if (N == 0) return SLA_OK;
  if (!x || !coords || !w_h || !w_w || !w_3 || !out || x == out) return SLA_ERR_INVALID_ARG;
  if (!aligned16(coords)) return SLA_ERR_UNSUPPORTED;
  if (!workspace || workspace_bytes < sla_cwi_workspace_bytes(batch, grid_z, grid_h, grid_w) || !aligned16(workspace))
    return SLA_ERR_WORKSPACE;
  cudaError_t e = sla::launch_cwi(x, coords, (int)N, C, dt, batch, grid_z, grid_h, grid_w, S_h, S_w, w_h, w_w, w_3, out,
                                  static_cast<int32_t*>(workspace),
                                  reinterpret_cast<uint32_t*>(static_cast<char*>(workspace) +
                                      ((size_t)cwi_cells(batch, grid_z, grid_h, grid_w) * 4 + 15) / 16 * 16),
                                  (cudaStream_t)stream);
  return e == cudaSuccess ? SLA_OK : SLA_ERR_CUDA;
}

int sla_bench_stream_ceiling(const void* a, const void* b, const void* c, void* out, size_t bytes,
                             sla_stream_t stream) {
  if (!a || !b || !c || !out) return SLA_ERR_INVALID_ARG;
  if (bytes % 16 != 0 || !aligned16(a) || !aligned16(b) || !aligned16(c) || !aligned16(out)) return SLA_ERR_UNSUPPORTED;
  cudaError_t e = sla::launch_stream_ceiling(a, b, c, out, bytes, (cudaStream_t)stream);
  return e == cudaSuccess ? SLA_OK : SLA_ERR_CUDA;
}

static int forward_impl(bool tcgen05, int phi, float eps, const void* q, const void* k, const void* v, const int32_t* window_offsets, int64_t N,
                        int32_t W, int32_t H, int32_t d_h, int dt, void* out, void* workspace,
                        size_t workspace_bytes, sla_stream_t stream) {
  int rc = check_common(N, W, H, d_h, dt);
  if (rc != SLA_OK) return rc;
  if (N == 0 || W == 0) return SLA_OK;
  if (!q || !k || !v || !window_offsets || !out) return SLA_ERR_INVALID_ARG;
  if (!aligned16(q) || !aligned16(k) || !aligned16(v) || !aligned16(out)) return SLA_ERR_UNSUPPORTED;
  const size_t need = state_bytes(N, H, d_h);
  if (!workspace || workspace_bytes < need || !aligned16(workspace)) return SLA_ERR_WORKSPACE;
  cudaStream_t st = (cudaStream_t)stream;
  if (sla::launch_zero(workspace, need, st) != cudaSuccess) return SLA_ERR_CUDA;
  sla::Problem p{};
  p.q = q; p.k = k; p.v = v; p.out = out; p.off = window_offsets;
  p.ws_state = static_cast<float*>(workspace);
  p.N = (int)N; p.W = W; p.H = H; p.d = d_h;
  p.tcgen05 = tcgen05;
  p.phi = phi; p.eps = eps;
  if (tcgen05 && !sla::forward_umma_supported(p, dt)) return SLA_ERR_UNSUPPORTED;
  const bool tc = sla::forward_tc_supported(p, dt);
  cudaError_t e = tc ? sla::launch_forward_tc(p, dt, st) : sla::launch_forward_generic(p, dt, st);
  return e == cudaSuccess ? SLA_OK : SLA_ERR_CUDA;
}

int sla_forward(const void* q, const void* k, const void* v, const int32_t* window_offsets, int64_t N,
                int32_t W, int32_t H, int32_t d_h, int dt, void* out, void* workspace,
                size_t workspace_bytes, sla_stream_t stream) {
  return forward_impl(false, SLA_PHI_ELU1, 0.f, q, k, v, window_offsets, N, W, H, d_h, dt, out, workspace, workspace_bytes, stream);
}

int sla_module_forward(const void* x, const void* w_qkv, const float* bias, const int32_t* window_offsets, int64_t N,
                       int32_t W, int32_t H, int32_t d_h, int dt, void* q, void* k, void* v, void* out,
                       void* workspace, size_t workspace_bytes, sla_stream_t stream) {
  int rc = check_common(N, W, H, d_h, dt);
  if (rc != SLA_OK) return rc;
  // projection, then the op on its results: the kernels follow each other on `stream` as one chain of programmatic
  // dependent launches, and q, k, v (3 N C elements) are still in L2 when the op reads them if they fit there
  rc = sla_qkv_projection(x, w_qkv, bias, N, H * d_h, dt, q, k, v, stream);
  if (rc != SLA_OK) return rc;
  return forward_impl(false, SLA_PHI_ELU1, 0.f, q, k, v, window_offsets, N, W, H, d_h, dt, out, workspace,
                      workspace_bytes, stream);
}

// feature map / epsilon arguments of the *_phi entries
static int check_phi(int phi, float eps) {
  if (phi != SLA_PHI_ELU1 && phi != SLA_PHI_RELU) return SLA_ERR_INVALID_ARG;
  if (!(eps >= 0.f) || (phi == SLA_PHI_ELU1 && eps != 0.f)) return SLA_ERR_INVALID_ARG;
  return SLA_OK;
}

int sla_forward_phi(const void* q, const void* k, const void* v, const int32_t* window_offsets, int64_t N,
                    int32_t W, int32_t H, int32_t d_h, int dt, int feature_map, float eps, void* out,
                    void* workspace, size_t workspace_bytes, sla_stream_t stream) {
  const int rc = check_phi(feature_map, eps);
  if (rc != SLA_OK) return rc;
  return forward_impl(false, feature_map, eps, q, k, v, window_offsets, N, W, H, d_h, dt, out, workspace,
                      workspace_bytes, stream);
}

int sla_forward_tcgen05(const void* q, const void* k, const void* v, const int32_t* window_offsets, int64_t N,
                        int32_t W, int32_t H, int32_t d_h, int dt, void* out, void* workspace,
                        size_t workspace_bytes, sla_stream_t stream) {
  return forward_impl(true, SLA_PHI_ELU1, 0.f, q, k, v, window_offsets, N, W, H, d_h, dt, out, workspace, workspace_bytes, stream);
}

int sla_forward_static(const void* q, const void* k, const void* v, const int32_t* window_offsets, int64_t N,
                       int32_t W, int32_t H, int32_t d_h, int dt, void* out, sla_stream_t stream) {
  const int rc = check_common(N, W, H, d_h, dt);
  if (rc != SLA_OK) return rc;
  if (N == 0 || W == 0) return SLA_OK;
  // what sla_forward would ask the caller for must fit the static array; checked before anything is launched
  if (state_bytes(N, H, d_h) > (size_t)SLA_STATIC_WORKSPACE_BYTES) return SLA_ERR_TOO_LARGE;
  void* ws = nullptr;
  const int rs = static_workspace(&ws);
  if (rs != SLA_OK) return rs;
  // from here on the general entry's own path (it zeroes the part of the workspace it uses on `stream` first): the
  // array keeps the previous call's contents, and two calls that overlap on the GPU would race on it
  return forward_impl(false, SLA_PHI_ELU1, 0.f, q, k, v, window_offsets, N, W, H, d_h, dt, out, ws,
                      (size_t)SLA_STATIC_WORKSPACE_BYTES, stream);
}

int sla_forward_bounded(const void* q, const void* k, const void* v, const int32_t* window_offsets,
                        int64_t N, int32_t W, int32_t H, int32_t d_h, int dt, void* out,
                        int32_t max_window_len, sla_stream_t stream) {
  int rc = check_common(N, W, H, d_h, dt);
  if (rc != SLA_OK) return rc;
  if (max_window_len < 1) return SLA_ERR_INVALID_ARG;
  if (max_window_len > sla::kFuseMax) return SLA_ERR_UNSUPPORTED;   // use sla_forward
  if (N == 0 || W == 0) return SLA_OK;
  if (!q || !k || !v || !window_offsets || !out) return SLA_ERR_INVALID_ARG;
  if (!aligned16(q) || !aligned16(k) || !aligned16(v) || !aligned16(out)) return SLA_ERR_UNSUPPORTED;
  sla::Problem p{};
  p.q = q; p.k = k; p.v = v; p.out = out; p.off = window_offsets;
  p.N = (int)N; p.W = W; p.H = H; p.d = d_h;
  p.bounded = true;                                           // one launch: no workspace, no split pass
  const bool tc = sla::forward_tc_supported(p, dt);
  cudaError_t e = tc ? sla::launch_forward_tc(p, dt, (cudaStream_t)stream)
                     : sla::launch_forward_generic(p, dt, (cudaStream_t)stream);
  return e == cudaSuccess ? SLA_OK : SLA_ERR_CUDA;
}

size_t sla_span_table_bytes(int64_t N, int32_t H, int32_t d_h) {
  if (N < 0 || N >= (int64_t(1) << 31) || H < 1 || (d_h != 16 && d_h != 32)) return 0;
  return sla::span_table_bytes(N, H, d_h);
}

int sla_build_span_table(const int32_t* window_offsets, int64_t N, int32_t W, int32_t H, int32_t d_h, void* table,
                         size_t table_bytes, sla_stream_t stream) {
  if (N < 0 || W < 0 || H < 1 || N >= (int64_t(1) << 31)) return SLA_ERR_INVALID_ARG;
  if (d_h != 16 && d_h != 32) return SLA_ERR_UNSUPPORTED;
  if (!table || table_bytes < sla::span_table_bytes(N, H, d_h) || !aligned16(table)) return SLA_ERR_WORKSPACE;
  if (N == 0 || W == 0) return SLA_OK;
  if (!window_offsets) return SLA_ERR_INVALID_ARG;
  cudaError_t e = sla::launch_span_table(window_offsets, (int)N, W, H, d_h, table, (cudaStream_t)stream);
  return e == cudaSuccess ? SLA_OK : SLA_ERR_CUDA;
}

int sla_forward_planned(const void* q, const void* k, const void* v, const int32_t* window_offsets, int64_t N,
                        int32_t W, int32_t H, int32_t d_h, int dt, void* out, int32_t max_window_len,
                        const void* table, size_t table_bytes, sla_stream_t stream) {
  int rc = check_common(N, W, H, d_h, dt);
  if (rc != SLA_OK) return rc;
  if (max_window_len < 1) return SLA_ERR_INVALID_ARG;
  if (max_window_len > sla::kFuseMax) return SLA_ERR_UNSUPPORTED;   // use sla_forward
  if (N == 0 || W == 0) return SLA_OK;
  if (!q || !k || !v || !window_offsets || !out) return SLA_ERR_INVALID_ARG;
  if (!aligned16(q) || !aligned16(k) || !aligned16(v) || !aligned16(out)) return SLA_ERR_UNSUPPORTED;
  if (!table || table_bytes < sla::span_table_bytes(N, H, d_h) || !aligned16(table)) return SLA_ERR_WORKSPACE;
  sla::Problem p{};
  p.q = q; p.k = k; p.v = v; p.out = out; p.off = window_offsets;
  p.N = (int)N; p.W = W; p.H = H; p.d = d_h;
  p.bounded = true;
  p.span_table = table;
  const bool tc = sla::forward_tc_supported(p, dt);           // the generic kernels have no use for the table
  cudaError_t e = tc ? sla::launch_forward_tc(p, dt, (cudaStream_t)stream)
                     : sla::launch_forward_generic(p, dt, (cudaStream_t)stream);
  return e == cudaSuccess ? SLA_OK : SLA_ERR_CUDA;
}

static int backward_impl(int phi, float eps, const void* q, const void* k, const void* v, const int32_t* window_offsets, int64_t N,
                 int32_t W, int32_t H, int32_t d_h, int dt, const void* d_out, void* dq, void* dk,
                 void* dv, void* workspace, size_t workspace_bytes, sla_stream_t stream) {
  int rc = check_common(N, W, H, d_h, dt);
  if (rc != SLA_OK) return rc;
  if (N == 0 || W == 0) return SLA_OK;
  if (!q || !k || !v || !window_offsets || !d_out || !dq || !dk || !dv) return SLA_ERR_INVALID_ARG;
  if (!aligned16(q) || !aligned16(k) || !aligned16(v) || !aligned16(d_out) || !aligned16(dq) ||
      !aligned16(dk) || !aligned16(dv))
    return SLA_ERR_UNSUPPORTED;
  const size_t one = state_bytes(N, H, d_h);
  if (!workspace || workspace_bytes < 2 * one || !aligned16(workspace)) return SLA_ERR_WORKSPACE;
  cudaStream_t st = (cudaStream_t)stream;
  if (sla::launch_zero(workspace, 2 * one, st) != cudaSuccess) return SLA_ERR_CUDA;
  sla::Problem p{};
  p.q = q; p.k = k; p.v = v; p.g = d_out; p.dq = dq; p.dk = dk; p.dv = dv; p.off = window_offsets;
  p.ws_state = static_cast<float*>(workspace);
  p.ws_dstate = reinterpret_cast<float*>(static_cast<char*>(workspace) + one);
  p.N = (int)N; p.W = W; p.H = H; p.d = d_h;
  p.phi = phi; p.eps = eps;
  const bool tc = sla::backward_tc_supported(p, dt);
  cudaError_t e = tc ? sla::launch_backward_tc(p, dt, st) : sla::launch_backward_generic(p, dt, st);
  return e == cudaSuccess ? SLA_OK : SLA_ERR_CUDA;
}

int sla_backward(const void* q, const void* k, const void* v, const int32_t* window_offsets, int64_t N,
                 int32_t W, int32_t H, int32_t d_h, int dt, const void* d_out, void* dq, void* dk,
                 void* dv, void* workspace, size_t workspace_bytes, sla_stream_t stream) {
  return backward_impl(SLA_PHI_ELU1, 0.f, q, k, v, window_offsets, N, W, H, d_h, dt, d_out, dq, dk, dv, workspace,
                       workspace_bytes, stream);
}

int sla_backward_bounded(const void* q, const void* k, const void* v, const int32_t* window_offsets, int64_t N,
                         int32_t W, int32_t H, int32_t d_h, int dt, const void* d_out, void* dq, void* dk, void* dv,
                         int32_t max_window_len, sla_stream_t stream) {
  int rc = check_common(N, W, H, d_h, dt);
  if (rc != SLA_OK) return rc;
  if (max_window_len < 1) return SLA_ERR_INVALID_ARG;
  if (max_window_len > sla::kFuseMax) return SLA_ERR_UNSUPPORTED;   // use sla_backward
  if (N == 0 || W == 0) return SLA_OK;
  if (!q || !k || !v || !window_offsets || !d_out || !dq || !dk || !dv) return SLA_ERR_INVALID_ARG;
  if (!aligned16(q) || !aligned16(k) || !aligned16(v) || !aligned16(d_out) || !aligned16(dq) ||
      !aligned16(dk) || !aligned16(dv))
    return SLA_ERR_UNSUPPORTED;
  sla::Problem p{};
  p.q = q; p.k = k; p.v = v; p.g = d_out; p.dq = dq; p.dk = dk; p.dv = dv; p.off = window_offsets;
  p.N = (int)N; p.W = W; p.H = H; p.d = d_h;
  p.phi = SLA_PHI_ELU1; p.eps = 0.f;
  p.bounded = true;                                           // one launch: no workspace, no split passes
  const bool tc = sla::backward_tc_supported(p, dt);
  cudaError_t e = tc ? sla::launch_backward_tc(p, dt, (cudaStream_t)stream)
                     : sla::launch_backward_generic(p, dt, (cudaStream_t)stream);
  return e == cudaSuccess ? SLA_OK : SLA_ERR_CUDA;
}

int sla_backward_phi(const void* q, const void* k, const void* v, const int32_t* window_offsets, int64_t N,
                     int32_t W, int32_t H, int32_t d_h, int dt, int feature_map, float eps, const void* d_out,
                     void* dq, void* dk, void* dv, void* workspace, size_t workspace_bytes, sla_stream_t stream) {
  const int rc = check_phi(feature_map, eps);
  if (rc != SLA_OK) return rc;
  return backward_impl(feature_map, eps, q, k, v, window_offsets, N, W, H, d_h, dt, d_out, dq, dk, dv, workspace,
                       workspace_bytes, stream);
}

}  // extern "C"

namespace {
// Memory pool of the host-buffer entry, one per device, created on first use and kept for the life of
// the process.  Its release threshold is unbounded, so the staging block of one call is reused by the
// next instead of going back to the driver at every stream synchronisation (the default pool's
// threshold is 0: a real allocation and free of ~80 MB per call, several ms).
cudaMemPool_t host_entry_pool() {
  static cudaMemPool_t pools[64] = {};
  static std::mutex mu;
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return nullptr;
  std::lock_guard<std::mutex> lock(mu);
  if (!pools[dev]) {
    cudaMemPoolProps props = {};
    props.allocType = cudaMemAllocationTypePinned;
    props.handleTypes = cudaMemHandleTypeNone;
    props.location.type = cudaMemLocationTypeDevice;
    props.location.id = dev;
    cudaMemPool_t pool = nullptr;
    if (cudaMemPoolCreate(&pool, &props) != cudaSuccess) { (void)cudaGetLastError(); return nullptr; }
    unsigned long long thr = ~0ull;
    cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &thr);
    pools[dev] = pool;
  }
  return pools[dev];
}
// Two copy streams per device for the host entry (host -> device, device -> host), created on first use and kept for the
// life of the process like the pool.  Work on them is ordered against the caller's stream with events only.
struct HostLanes { cudaStream_t in, out; };
HostLanes* host_entry_lanes() {
  static HostLanes lanes[64] = {};
  static bool made[64] = {};
  static std::mutex mu;
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return nullptr;
  std::lock_guard<std::mutex> lock(mu);
  if (!made[dev]) {
    if (cudaStreamCreateWithFlags(&lanes[dev].in, cudaStreamNonBlocking) != cudaSuccess ||
        cudaStreamCreateWithFlags(&lanes[dev].out, cudaStreamNonBlocking) != cudaSuccess) {
      (void)cudaGetLastError();
      return nullptr;
    }
    made[dev] = true;
  }
  return &lanes[dev];
}
}  // namespace

extern "C" {

int sla_forward_host(const void* q, const void* k, const void* v, const int32_t* win_id, int64_t N,
                     int32_t W, int32_t H, int32_t d_h, int dt, void* out, sla_stream_t stream) {
  int rc = check_common(N, W, H, d_h, dt);
  if (rc != SLA_OK) return rc;
  if (N == 0 || W == 0) return SLA_OK;
  if (!q || !k || !v || !win_id || !out) return SLA_ERR_INVALID_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  const size_t row = (size_t)H * d_h * esize(dt);              // bytes per row of one tensor
  const size_t tb = (size_t)N * row;
  const size_t tb_al = (tb + 255) / 256 * 256;
  const size_t ids_al = ((size_t)N * 4 + 255) / 256 * 256;
  // The scene is cut at window boundaries into up to kHostChunks chunks of about equal row count (host-side scan of the
  // ids, integers only).  Chunk c+1 travels host -> device while chunk c is computed and chunk c-1 travels back: the two
  // directions of the link are independent, so the copy out hides behind the copy in.
  constexpr int kHostChunks = 4;
  int64_t cut[kHostChunks + 1];
  int nch = 0;
  cut[0] = 0;
  const int want = N >= 16384 ? kHostChunks : 1;
  for (int c = 1; c < want; ++c) {
    int64_t r = N * c / want;
    if (r <= cut[nch]) continue;
    while (r < N && win_id[r] == win_id[r - 1]) ++r;           // move the cut to the next window boundary
    if (r >= N) break;
    cut[++nch] = r;
  }
  cut[++nch] = N;
  size_t off_al = 0;                                           // local offsets of all chunks, back to back
  int32_t w0[kHostChunks], wc[kHostChunks];
  for (int c = 0; c < nch; ++c) {
    w0[c] = win_id[cut[c]];
    wc[c] = win_id[cut[c + 1] - 1] - w0[c] + 1;
    if (w0[c] < 0 || wc[c] < 1 || (int64_t)w0[c] + wc[c] > W) return SLA_ERR_INVALID_ARG;   // ids not sorted in [0, W)
    off_al += ((size_t)(wc[c] + 1) * 4 + 255) / 256 * 256;
  }
  const size_t ws = state_bytes(N, H, d_h);
  HostLanes* lanes = host_entry_lanes();
  cudaMemPool_t pool = host_entry_pool();
  if (!lanes) return SLA_ERR_CUDA;
  char* base = nullptr;
  const size_t total = 4 * tb_al + ids_al + off_al + ws;
  const cudaError_t ae = pool ? cudaMallocFromPoolAsync(reinterpret_cast<void**>(&base), total, pool, st)
                              : cudaMallocAsync(reinterpret_cast<void**>(&base), total, st);
  if (ae != cudaSuccess) return SLA_ERR_CUDA;
  char* dq_ = base; char* dk_ = base + tb_al; char* dv_ = base + 2 * tb_al; char* do_ = base + 3 * tb_al;
  int32_t* dids = reinterpret_cast<int32_t*>(base + 4 * tb_al);
  char* doff = base + 4 * tb_al + ids_al;
  void* dws = base + 4 * tb_al + ids_al + off_al;
  cudaEvent_t ev_start = nullptr, ev_in[kHostChunks] = {}, ev_done[kHostChunks] = {}, ev_out = nullptr;
  bool ok = cudaEventCreateWithFlags(&ev_start, cudaEventDisableTiming) == cudaSuccess &&
            cudaEventCreateWithFlags(&ev_out, cudaEventDisableTiming) == cudaSuccess;
  for (int c = 0; c < nch && ok; ++c)
    ok = cudaEventCreateWithFlags(&ev_in[c], cudaEventDisableTiming) == cudaSuccess &&
         cudaEventCreateWithFlags(&ev_done[c], cudaEventDisableTiming) == cudaSuccess;
  // the copy lanes start after whatever precedes this call on the caller's stream (and after the allocation)
  ok = ok && cudaEventRecord(ev_start, st) == cudaSuccess && cudaStreamWaitEvent(lanes->in, ev_start, 0) == cudaSuccess &&
       cudaStreamWaitEvent(lanes->out, ev_start, 0) == cudaSuccess;
  for (int c = 0; c < nch && ok; ++c) {                        // lane "in": host -> device, chunk by chunk
    const int64_t r0 = cut[c], n = cut[c + 1] - cut[c];
    ok = ok && cudaMemcpyAsync(dids + r0, win_id + r0, (size_t)n * 4, cudaMemcpyHostToDevice, lanes->in) == cudaSuccess;
    ok = ok && cudaMemcpyAsync(dk_ + r0 * row, (const char*)k + r0 * row, n * row, cudaMemcpyHostToDevice, lanes->in) == cudaSuccess;
    ok = ok && cudaMemcpyAsync(dv_ + r0 * row, (const char*)v + r0 * row, n * row, cudaMemcpyHostToDevice, lanes->in) == cudaSuccess;
    ok = ok && cudaMemcpyAsync(dq_ + r0 * row, (const char*)q + r0 * row, n * row, cudaMemcpyHostToDevice, lanes->in) == cudaSuccess;
    ok = ok && cudaEventRecord(ev_in[c], lanes->in) == cudaSuccess;
  }
  size_t off_pos = 0;
  for (int c = 0; c < nch && ok && rc == SLA_OK; ++c) {        // caller's stream: prep + forward of chunk c
    const int64_t r0 = cut[c], n = cut[c + 1] - cut[c];
    int32_t* off_c = reinterpret_cast<int32_t*>(doff + off_pos);
    off_pos += ((size_t)(wc[c] + 1) * 4 + 255) / 256 * 256;
    ok = ok && cudaStreamWaitEvent(st, ev_in[c], 0) == cudaSuccess;
    ok = ok && sla::launch_offsets(dids + r0, (int)n, wc[c], off_c, st, w0[c]) == cudaSuccess;
    if (ok) rc = sla_forward(dq_ + r0 * row, dk_ + r0 * row, dv_ + r0 * row, off_c, n, wc[c], H, d_h, dt, do_ + r0 * row,
                             dws, ws, stream);
    ok = ok && cudaEventRecord(ev_done[c], st) == cudaSuccess;
    // lane "out": device -> host as soon as the chunk is done
    ok = ok && cudaStreamWaitEvent(lanes->out, ev_done[c], 0) == cudaSuccess;
    ok = ok && cudaMemcpyAsync((char*)out + r0 * row, do_ + r0 * row, n * row, cudaMemcpyDeviceToHost, lanes->out) == cudaSuccess;
  }
  // join the lanes back into the caller's stream before the block goes back to the pool
  if (ev_out && cudaEventRecord(ev_out, lanes->out) == cudaSuccess) cudaStreamWaitEvent(st, ev_out, 0);
  else cudaStreamSynchronize(lanes->out);
  if (ev_start && cudaEventRecord(ev_start, lanes->in) == cudaSuccess) cudaStreamWaitEvent(st, ev_start, 0);
  else cudaStreamSynchronize(lanes->in);
  cudaFreeAsync(base, st);
  if (cudaStreamSynchronize(st) != cudaSuccess) ok = false;
  if (ev_start) cudaEventDestroy(ev_start);
  if (ev_out) cudaEventDestroy(ev_out);
  for (int c = 0; c < kHostChunks; ++c) {
    if (ev_in[c]) cudaEventDestroy(ev_in[c]);
    if (ev_done[c]) cudaEventDestroy(ev_done[c]);
  }
  if (rc != SLA_OK) return rc;
  return ok ? SLA_OK : SLA_ERR_CUDA;
}

}  // extern "C"
