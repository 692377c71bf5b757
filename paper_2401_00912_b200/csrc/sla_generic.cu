// sla_generic.cu -- generic SLA forward/backward on the CUDA cores with fp32 arithmetic.
//
// This is the path for (a) fp32 I/O (tolerance 1e-5 rules out fp16/tf32 tensor-core operands) and
// (b) every shape/dtype the tensor-core path does not take.  It is load-balanced by fixed chunks of
// the flat sequence, not by window (Fig. 3a "chunks of uniform length"):
//
//   * thread block t owns TILE_ROWS consecutive rows [t*L,(t+1)*L) of the flat, window-sorted matrix;
//   * a window of <= FUSE_MAX rows is processed WHOLE by the block owning its first row: the state
//     S_w (d x d) and z_w (d) of Eq. 3 live in registers, the output pass follows in
//     the same block, nothing is written but `out`;
//   * a longer window is split at tile boundaries; each piece adds its partial state to an fp32
//     accumulator in the workspace (segmented reduction across chunks, red.global.add.f32) and a
//     second stream-ordered kernel emits the outputs of those pieces.
//
// Thread mapping: one thread per channel c = h*d + x.  The thread keeps column x of S_h
// (S[0..d-1][x], d registers) and z[x].  phi(k) / phi(q) of a staged row are broadcast through
// shared memory (each of the d threads of a head reads the head's d values with LDS.128).
#include "sla_internal.cuh"

namespace sla {
namespace {

constexpr int RB = kRowBatch;

template <int D>
__device__ __forceinline__ float reduce_head(float x) {  // sum over the D lanes of one head
#pragma unroll
  for (int o = D / 2; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
  return x;
}

struct Ctx {
  int C;       // H*d channels per row
  int c;       // this thread's channel (valid if active)
  int hl;      // local head index inside the block
  int x;       // channel inside the head
  int CB;      // threads per block
  bool active; // h < H
  bool relu;   // feature map: false = elu(x)+1, true = max(x,0)
  float eps;   // added to the denominator of Eq. 3 (0 for elu+1)
};

// S[p] += sum_j phi(k_j[h][p]) * v_j[h][x] ; z += sum_j phi(k_j[h][x])   over rows [r0,r1)
template <typename T, int D>
__device__ __forceinline__ void accumulate_state(const T* __restrict__ k, const T* __restrict__ v,
                                                 int r0, int r1, const Ctx& cx, float* bs,
                                                 float (&S)[D], float& z) {
  for (int base = r0; base < r1; base += RB) {
    const int nb = min(RB, r1 - base);
    float vv[RB];
#pragma unroll
    for (int i = 0; i < RB; ++i) {
      vv[i] = 0.f;
      if (i < nb && cx.active) {
        const size_t idx = (size_t)(base + i) * cx.C + cx.c;
        const float b = phi_f32(Elem<T>::ld(k + idx), cx.relu);
        vv[i] = Elem<T>::ld(v + idx);
        bs[i * cx.CB + threadIdx.x] = b;
        z += b;
      }
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < RB; ++i) {
      if (i < nb) {
        const float4* bp = reinterpret_cast<const float4*>(bs + i * cx.CB + cx.hl * D);
#pragma unroll
        for (int p4 = 0; p4 < D / 4; ++p4) {
          const float4 b4 = bp[p4];
          S[4 * p4 + 0] = fmaf(b4.x, vv[i], S[4 * p4 + 0]);
          S[4 * p4 + 1] = fmaf(b4.y, vv[i], S[4 * p4 + 1]);
          S[4 * p4 + 2] = fmaf(b4.z, vv[i], S[4 * p4 + 2]);
          S[4 * p4 + 3] = fmaf(b4.w, vv[i], S[4 * p4 + 3]);
        }
      }
    }
    __syncthreads();
  }
}

// out_i[h][x] = sum_p phi(q_i[h][p]) S[p][x] / sum_p phi(q_i[h][p]) z[p]     rows [r0,r1)
template <typename T, int D>
__device__ __forceinline__ void emit_output(const T* __restrict__ q, T* __restrict__ out, int r0,
                                            int r1, const Ctx& cx, float* bs, const float (&S)[D],
                                            float z) {
  for (int base = r0; base < r1; base += RB) {
    const int nb = min(RB, r1 - base);
    float aown[RB];
#pragma unroll
    for (int i = 0; i < RB; ++i) {
      aown[i] = 0.f;
      if (i < nb && cx.active) {
        aown[i] = phi_f32(Elem<T>::ld(q + (size_t)(base + i) * cx.C + cx.c), cx.relu);
        bs[i * cx.CB + threadIdx.x] = aown[i];
      }
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < RB; ++i) {
      if (i < nb) {
        const float4* ap = reinterpret_cast<const float4*>(bs + i * cx.CB + cx.hl * D);
        float num = 0.f;
#pragma unroll
        for (int p4 = 0; p4 < D / 4; ++p4) {
          const float4 a4 = ap[p4];
          num = fmaf(a4.x, S[4 * p4 + 0], num);
          num = fmaf(a4.y, S[4 * p4 + 1], num);
          num = fmaf(a4.z, S[4 * p4 + 2], num);
          num = fmaf(a4.w, S[4 * p4 + 3], num);
        }
        const float den = reduce_head<D>(aown[i] * z) + cx.eps;
        if (cx.active) Elem<T>::st(out + (size_t)(base + i) * cx.C + cx.c, num / den);
      }
    }
    __syncthreads();
  }
}

template <int D>
__device__ __forceinline__ float* state_slot(float* ws, int s, int H, int h) {
  // A split window has > kFuseMax rows, so floor(s/(kFuseMax+1)) of its first row s is unique to it.
  return ws + kWsHeaderFloats + ((size_t)(s / (kFuseMax + 1)) * H + h) * (size_t)((D + 1) * D);
}

__device__ __forceinline__ Ctx make_ctx(int H, int D, bool relu, float eps) {
  Ctx cx;
  cx.relu = relu;   // a compile-time constant of the calling kernel: the feature-map branches fold away
  cx.eps = eps;
  cx.CB = blockDim.x;
  const int HB = cx.CB / D;
  cx.hl = threadIdx.x / D;
  cx.x = threadIdx.x % D;
  const int h = blockIdx.y * HB + cx.hl;
  cx.active = h < H;
  cx.C = H * D;
  cx.c = h * D + cx.x;
  return cx;
}

// ------------------------------------------------------------------------------------------------
// Forward, main kernel: fused whole windows + partial states of split windows.
template <typename T, int D, bool RELU>
__global__ void __launch_bounds__(256)
sla_fwd_generic_kernel(const T* __restrict__ q, const T* __restrict__ k, const T* __restrict__ v,
                       const int32_t* __restrict__ off, T* __restrict__ out, float* __restrict__ ws,
                       int N, int W, int H, float eps) {
  __shared__ __align__(16) float bs[RB * 256];
  const Ctx cx = make_ctx(H, D, RELU, eps);
  const int h = cx.c / D;
  const int row0 = blockIdx.x * kTileRows;
  const int row1 = min(row0 + kTileRows, N);
  for (int w = window_of_row(off, W, row0); w < W; ++w) {
    const int s = __ldg(off + w), e = __ldg(off + w + 1);
    if (s >= row1) break;
    const int m = e - s;
    if (m <= 0) continue;
    if (m <= kFuseMax) {
      if (s < row0) continue;  // owned by the tile that holds its first row
      float S[D], z = 0.f;
#pragma unroll
      for (int p = 0; p < D; ++p) S[p] = 0.f;
      accumulate_state<T, D>(k, v, s, e, cx, bs, S, z);
      emit_output<T, D>(q, out, s, e, cx, bs, S, z);
    } else if (ws != nullptr) {   // bounded entry (no workspace): a window that breaks the caller's promise is skipped
      float S[D], z = 0.f;
#pragma unroll
      for (int p = 0; p < D; ++p) S[p] = 0.f;
      accumulate_state<T, D>(k, v, max(s, row0), min(e, row1), cx, bs, S, z);
      if (threadIdx.x == 0) reinterpret_cast<volatile int*>(ws)[0] = 1;
      if (cx.active) {
        float* slot = state_slot<D>(ws, s, H, h);
#pragma unroll
        for (int p = 0; p < D; ++p) atomicAdd(slot + p * D + cx.x, S[p]);
        atomicAdd(slot + D * D + cx.x, z);
      }
    }
  }
}

// Forward, second kernel: outputs of the pieces of split windows (state read from the workspace).
template <typename T, int D, bool RELU>
__global__ void __launch_bounds__(256)
sla_fwd_generic_split_kernel(const T* __restrict__ q, const int32_t* __restrict__ off,
                             T* __restrict__ out, const float* __restrict__ ws, int N, int W, int H, float eps) {
  __shared__ __align__(16) float bs[RB * 256];
  if (reinterpret_cast<const volatile int*>(ws)[0] == 0) return;   // no split window in this call
  const Ctx cx = make_ctx(H, D, RELU, eps);
  const int h = cx.c / D;
  const int row0 = blockIdx.x * kTileRows;
  const int row1 = min(row0 + kTileRows, N);
  for (int w = window_of_row(off, W, row0); w < W; ++w) {
    const int s = __ldg(off + w), e = __ldg(off + w + 1);
    if (s >= row1) break;
    if (e - s <= kFuseMax) continue;
    float S[D], z = 0.f;
#pragma unroll
    for (int p = 0; p < D; ++p) S[p] = 0.f;
    if (cx.active) {
      const float* slot = state_slot<D>(const_cast<float*>(ws), s, H, h);
#pragma unroll
      for (int p = 0; p < D; ++p) S[p] = slot[p * D + cx.x];
      z = slot[D * D + cx.x];
    }
    emit_output<T, D>(q, out, max(s, row0), min(e, row1), cx, bs, S, z);
  }
}

// ------------------------------------------------------------------------------------------------
// Backward (derivatives of Eq. 3; the paper is silent on training).
// Thread (h,x) holds column x of S and of dS ("col": X[p][x]) and row x of S / dS ("row": X[x][r]).
constexpr int TB_PITCH_EXTRA = 1;

// col -> row transpose of a per-head d x d matrix through shared memory.
template <int D>
__device__ __forceinline__ void transpose_state(const float (&col)[D], float (&row)[D], const Ctx& cx,
                                                float* tb) {
  float* t = tb + cx.hl * D * (D + TB_PITCH_EXTRA);
  __syncthreads();
#pragma unroll
  for (int p = 0; p < D; ++p) t[p * (D + TB_PITCH_EXTRA) + cx.x] = col[p];
  __syncthreads();
#pragma unroll
  for (int r = 0; r < D; ++r) row[r] = t[cx.x * (D + TB_PITCH_EXTRA) + r];
  __syncthreads();
}

// Stage B2 over rows [r0,r1): dq, and accumulation of dS (column x) and dz[x].
//   dnum_i = g_i/den_i ; dden_i = -(g_i.o_i)/den_i ; da_i = dnum_i S^T + dden_i z ; dq_i = da_i*phi'(q_i)
//   dS += a_i^T dnum_i ; dz += dden_i a_i
template <typename T, int D>
__device__ __forceinline__ void backward_query_pass(const T* __restrict__ q, const T* __restrict__ g,
                                                    T* __restrict__ dq, int r0, int r1, const Ctx& cx,
                                                    float* bsA, float* bsB, const float (&Scol)[D],
                                                    const float (&Srow)[D], float z,
                                                    float (&dScol)[D], float& dz) {
  constexpr int RB2 = 4;
  for (int base = r0; base < r1; base += RB2) {
    const int nb = min(RB2, r1 - base);
    float qv[RB2], gv[RB2], aown[RB2], dnum[RB2], dden[RB2];
#pragma unroll
    for (int i = 0; i < RB2; ++i) {
      qv[i] = 0.f; gv[i] = 0.f; aown[i] = 0.f;
      if (i < nb && cx.active) {
        const size_t idx = (size_t)(base + i) * cx.C + cx.c;
        qv[i] = Elem<T>::ld(q + idx);
        gv[i] = Elem<T>::ld(g + idx);
        aown[i] = phi_f32(qv[i], cx.relu);
        bsA[i * cx.CB + threadIdx.x] = aown[i];
      }
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < RB2; ++i) {
      dnum[i] = 0.f; dden[i] = 0.f;
      if (i < nb) {
        const float4* ap = reinterpret_cast<const float4*>(bsA + i * cx.CB + cx.hl * D);
        float num = 0.f;
#pragma unroll
        for (int p4 = 0; p4 < D / 4; ++p4) {
          const float4 a4 = ap[p4];
          num = fmaf(a4.x, Scol[4 * p4 + 0], num);
          num = fmaf(a4.y, Scol[4 * p4 + 1], num);
          num = fmaf(a4.z, Scol[4 * p4 + 2], num);
          num = fmaf(a4.w, Scol[4 * p4 + 3], num);
        }
        const float den = reduce_head<D>(aown[i] * z) + cx.eps;
        const float inv = 1.f / den;
        const float o = num * inv;
        const float go = reduce_head<D>(gv[i] * o);
        dnum[i] = gv[i] * inv;
        dden[i] = -go * inv;
        if (cx.active) bsB[i * cx.CB + threadIdx.x] = dnum[i];
      }
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < RB2; ++i) {
      if (i < nb) {
        const float4* ap = reinterpret_cast<const float4*>(bsA + i * cx.CB + cx.hl * D);
        const float4* np = reinterpret_cast<const float4*>(bsB + i * cx.CB + cx.hl * D);
        float da = dden[i] * z;
#pragma unroll
        for (int p4 = 0; p4 < D / 4; ++p4) {
          const float4 n4 = np[p4];
          da = fmaf(n4.x, Srow[4 * p4 + 0], da);
          da = fmaf(n4.y, Srow[4 * p4 + 1], da);
          da = fmaf(n4.z, Srow[4 * p4 + 2], da);
          da = fmaf(n4.w, Srow[4 * p4 + 3], da);
          const float4 a4 = ap[p4];
          dScol[4 * p4 + 0] = fmaf(a4.x, dnum[i], dScol[4 * p4 + 0]);
          dScol[4 * p4 + 1] = fmaf(a4.y, dnum[i], dScol[4 * p4 + 1]);
          dScol[4 * p4 + 2] = fmaf(a4.z, dnum[i], dScol[4 * p4 + 2]);
          dScol[4 * p4 + 3] = fmaf(a4.w, dnum[i], dScol[4 * p4 + 3]);
        }
        dz = fmaf(dden[i], aown[i], dz);
        if (cx.active)
          Elem<T>::st(dq + (size_t)(base + i) * cx.C + cx.c, da * dphi_f32(qv[i], cx.relu));
      }
    }
    __syncthreads();
  }
}

// Stage B3 over rows [r0,r1): dk_j = (v_j dS^T + dz) * phi'(k_j) ; dv_j = b_j dS.
template <typename T, int D>
__device__ __forceinline__ void backward_key_pass(const T* __restrict__ k, const T* __restrict__ v,
                                                  T* __restrict__ dk, T* __restrict__ dv, int r0,
                                                  int r1, const Ctx& cx, float* bsA, float* bsB,
                                                  const float (&dScol)[D], const float (&dSrow)[D],
                                                  float dz) {
  constexpr int RB2 = 4;
  for (int base = r0; base < r1; base += RB2) {
    const int nb = min(RB2, r1 - base);
    float kv[RB2];
#pragma unroll
    for (int i = 0; i < RB2; ++i) {
      kv[i] = 0.f;
      if (i < nb && cx.active) {
        const size_t idx = (size_t)(base + i) * cx.C + cx.c;
        kv[i] = Elem<T>::ld(k + idx);
        bsA[i * cx.CB + threadIdx.x] = phi_f32(kv[i], cx.relu);
        bsB[i * cx.CB + threadIdx.x] = Elem<T>::ld(v + idx);
      }
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < RB2; ++i) {
      if (i < nb) {
        const float4* bp = reinterpret_cast<const float4*>(bsA + i * cx.CB + cx.hl * D);
        const float4* vp = reinterpret_cast<const float4*>(bsB + i * cx.CB + cx.hl * D);
        float dvx = 0.f, db = dz;
#pragma unroll
        for (int p4 = 0; p4 < D / 4; ++p4) {
          const float4 b4 = bp[p4];
          dvx = fmaf(b4.x, dScol[4 * p4 + 0], dvx);
          dvx = fmaf(b4.y, dScol[4 * p4 + 1], dvx);
          dvx = fmaf(b4.z, dScol[4 * p4 + 2], dvx);
          dvx = fmaf(b4.w, dScol[4 * p4 + 3], dvx);
          const float4 v4 = vp[p4];
          db = fmaf(v4.x, dSrow[4 * p4 + 0], db);
          db = fmaf(v4.y, dSrow[4 * p4 + 1], db);
          db = fmaf(v4.z, dSrow[4 * p4 + 2], db);
          db = fmaf(v4.w, dSrow[4 * p4 + 3], db);
        }
        if (cx.active) {
          const size_t idx = (size_t)(base + i) * cx.C + cx.c;
          Elem<T>::st(dv + idx, dvx);
          Elem<T>::st(dk + idx, db * dphi_f32(kv[i], cx.relu));
        }
      }
    }
    __syncthreads();
  }
}

template <int D> struct BwdSmem {
  static constexpr int kTb = (256 / D) * D * (D + TB_PITCH_EXTRA);
  static constexpr int kBs = 2 * RB * 256;
  static constexpr int kFloats = kTb > kBs ? kTb : kBs;
};

// Backward kernel 1: whole (fused) windows completely; partial states of split windows.
template <typename T, int D, bool RELU>
__global__ void __launch_bounds__(256, 2)
sla_bwd_generic_kernel(const T* __restrict__ q, const T* __restrict__ k, const T* __restrict__ v,
                       const T* __restrict__ g, const int32_t* __restrict__ off, T* __restrict__ dq,
                       T* __restrict__ dk, T* __restrict__ dv, float* __restrict__ ws, int N, int W,
                       int H, int split_only, float eps) {
  __shared__ __align__(16) float sm[BwdSmem<D>::kFloats];
  float* bsA = sm;
  float* bsB = sm + RB * 256;
  // split_only: the tensor-core kernel did every window <= kFuseMax rows and raised the workspace flag
  // if it met a longer one; here only those longer windows are accumulated
  if (split_only && reinterpret_cast<const volatile int*>(ws)[0] == 0) return;
  const Ctx cx = make_ctx(H, D, RELU, eps);
  const int h = cx.c / D;
  const int row0 = blockIdx.x * kBwdTileRows;
  const int row1 = min(row0 + kBwdTileRows, N);
  for (int w = window_of_row(off, W, row0); w < W; ++w) {
    const int s = __ldg(off + w), e = __ldg(off + w + 1);
    if (s >= row1) break;
    const int m = e - s;
    if (m <= 0) continue;
    float Scol[D], z = 0.f;
#pragma unroll
    for (int p = 0; p < D; ++p) Scol[p] = 0.f;
    if (m <= kFuseMax) {
      if (s < row0 || split_only) continue;
      accumulate_state<T, D>(k, v, s, e, cx, bsA, Scol, z);
      float Srow[D], dScol[D], dz = 0.f;
      transpose_state<D>(Scol, Srow, cx, sm);
#pragma unroll
      for (int p = 0; p < D; ++p) dScol[p] = 0.f;
      backward_query_pass<T, D>(q, g, dq, s, e, cx, bsA, bsB, Scol, Srow, z, dScol, dz);
      float dSrow[D];
      transpose_state<D>(dScol, dSrow, cx, sm);
      backward_key_pass<T, D>(k, v, dk, dv, s, e, cx, bsA, bsB, dScol, dSrow, dz);
    } else {
      if (ws == nullptr) continue;   // bounded entry (no workspace): a window that breaks the caller's promise is skipped
      accumulate_state<T, D>(k, v, max(s, row0), min(e, row1), cx, bsA, Scol, z);
      if (threadIdx.x == 0) reinterpret_cast<volatile int*>(ws)[0] = 1;
      if (cx.active) {
        float* slot = state_slot<D>(ws, s, H, h);
#pragma unroll
        for (int p = 0; p < D; ++p) atomicAdd(slot + p * D + cx.x, Scol[p]);
        atomicAdd(slot + D * D + cx.x, z);
      }
    }
  }
}

// Backward kernel 2 (split windows only): dq of each piece, dS/dz partials into the workspace.
template <typename T, int D, bool RELU>
__global__ void __launch_bounds__(256)
sla_bwd_generic_split_q_kernel(const T* __restrict__ q, const T* __restrict__ g,
                               const int32_t* __restrict__ off, T* __restrict__ dq,
                               const float* __restrict__ ws, float* __restrict__ wd, int N, int W,
                               int H, float eps) {
  __shared__ __align__(16) float sm[2 * RB * 256];
  float* bsA = sm;
  float* bsB = sm + RB * 256;
  if (reinterpret_cast<const volatile int*>(ws)[0] == 0) return;   // no split window in this call
  const Ctx cx = make_ctx(H, D, RELU, eps);
  const int h = cx.c / D;
  const int row0 = blockIdx.x * kBwdTileRows;
  const int row1 = min(row0 + kBwdTileRows, N);
  for (int w = window_of_row(off, W, row0); w < W; ++w) {
    const int s = __ldg(off + w), e = __ldg(off + w + 1);
    if (s >= row1) break;
    if (e - s <= kFuseMax) continue;
    float Scol[D], Srow[D], dScol[D], z = 0.f, dz = 0.f;
#pragma unroll
    for (int p = 0; p < D; ++p) { Scol[p] = 0.f; Srow[p] = 0.f; dScol[p] = 0.f; }
    if (cx.active) {
      const float* slot = state_slot<D>(const_cast<float*>(ws), s, H, h);
#pragma unroll
      for (int p = 0; p < D; ++p) { Scol[p] = slot[p * D + cx.x]; Srow[p] = slot[cx.x * D + p]; }
      z = slot[D * D + cx.x];
    }
    backward_query_pass<T, D>(q, g, dq, max(s, row0), min(e, row1), cx, bsA, bsB, Scol, Srow, z,
                              dScol, dz);
    if (cx.active) {
      float* slot = state_slot<D>(wd, s, H, h);
#pragma unroll
      for (int p = 0; p < D; ++p) atomicAdd(slot + p * D + cx.x, dScol[p]);
      atomicAdd(slot + D * D + cx.x, dz);
    }
  }
}

// Backward kernel 3 (split windows only): dk, dv of each piece.
template <typename T, int D, bool RELU>
__global__ void __launch_bounds__(256)
sla_bwd_generic_split_kv_kernel(const T* __restrict__ k, const T* __restrict__ v,
                                const int32_t* __restrict__ off, T* __restrict__ dk,
                                T* __restrict__ dv, const float* __restrict__ wd,
                                const float* __restrict__ ws, int N, int W, int H, float eps) {
  __shared__ __align__(16) float sm[2 * RB * 256];
  float* bsA = sm;
  float* bsB = sm + RB * 256;
  if (reinterpret_cast<const volatile int*>(ws)[0] == 0) return;   // no split window in this call
  const Ctx cx = make_ctx(H, D, RELU, eps);
  const int h = cx.c / D;
  const int row0 = blockIdx.x * kBwdTileRows;
  const int row1 = min(row0 + kBwdTileRows, N);
  for (int w = window_of_row(off, W, row0); w < W; ++w) {
    const int s = __ldg(off + w), e = __ldg(off + w + 1);
    if (s >= row1) break;
    if (e - s <= kFuseMax) continue;
    float dScol[D], dSrow[D], dz = 0.f;
#pragma unroll
    for (int p = 0; p < D; ++p) { dScol[p] = 0.f; dSrow[p] = 0.f; }
    if (cx.active) {
      const float* slot = state_slot<D>(const_cast<float*>(wd), s, H, h);
#pragma unroll
      for (int p = 0; p < D; ++p) { dScol[p] = slot[p * D + cx.x]; dSrow[p] = slot[cx.x * D + p]; }
      dz = slot[D * D + cx.x];
    }
    backward_key_pass<T, D>(k, v, dk, dv, max(s, row0), min(e, row1), cx, bsA, bsB, dScol, dSrow, dz);
  }
}

// ---- host-side dispatch -----------------------------------------------------------------------
inline int block_threads(int H, int D) {
  int c = H * D;
  c = (c + 31) / 32 * 32;
  return c < 256 ? c : 256;
}

template <typename T, int D, bool RELU>
cudaError_t fwd_launch(const Problem& p, cudaStream_t st) {
  const int CB = block_threads(p.H, D);
  const int HB = CB / D;
  dim3 grid((p.N + kTileRows - 1) / kTileRows, (p.H + HB - 1) / HB);
  sla_fwd_generic_kernel<T, D, RELU><<<grid, CB, 0, st>>>((const T*)p.q, (const T*)p.k, (const T*)p.v, p.off,
                                                    (T*)p.out, p.ws_state, p.N, p.W, p.H, p.eps);
  if (!p.bounded)
    sla_fwd_generic_split_kernel<T, D, RELU><<<grid, CB, 0, st>>>((const T*)p.q, p.off, (T*)p.out, p.ws_state,
                                                            p.N, p.W, p.H, p.eps);
  return cudaGetLastError();
}

template <typename T, int D, bool RELU>
cudaError_t bwd_launch(const Problem& p, cudaStream_t st, int split_only = 0) {
  const int CB = block_threads(p.H, D);
  const int HB = CB / D;
  dim3 grid((p.N + kBwdTileRows - 1) / kBwdTileRows, (p.H + HB - 1) / HB);
  sla_bwd_generic_kernel<T, D, RELU><<<grid, CB, 0, st>>>((const T*)p.q, (const T*)p.k, (const T*)p.v,
                                                    (const T*)p.g, p.off, (T*)p.dq, (T*)p.dk, (T*)p.dv,
                                                    p.ws_state, p.N, p.W, p.H, split_only, p.eps);
  if (p.bounded) return cudaGetLastError();   // no window is left to the split kernels
  sla_bwd_generic_split_q_kernel<T, D, RELU><<<grid, CB, 0, st>>>((const T*)p.q, (const T*)p.g, p.off,
                                                            (T*)p.dq, p.ws_state, p.ws_dstate, p.N, p.W,
                                                            p.H, p.eps);
  sla_bwd_generic_split_kv_kernel<T, D, RELU><<<grid, CB, 0, st>>>((const T*)p.k, (const T*)p.v, p.off,
                                                             (T*)p.dk, (T*)p.dv, p.ws_dstate, p.ws_state, p.N,
                                                             p.W, p.H, p.eps);
  return cudaGetLastError();
}

}  // namespace

cudaError_t launch_forward_generic(const Problem& p, int dt, cudaStream_t st) {
  if (p.d == 16) {
    if (dt == SLA_F32) return p.phi == SLA_PHI_RELU ? fwd_launch<float, 16, true>(p, st) : fwd_launch<float, 16, false>(p, st);
    if (dt == SLA_F16) return p.phi == SLA_PHI_RELU ? fwd_launch<__half, 16, true>(p, st) : fwd_launch<__half, 16, false>(p, st);
    return p.phi == SLA_PHI_RELU ? fwd_launch<__nv_bfloat16, 16, true>(p, st) : fwd_launch<__nv_bfloat16, 16, false>(p, st);
  }
  if (dt == SLA_F32) return p.phi == SLA_PHI_RELU ? fwd_launch<float, 32, true>(p, st) : fwd_launch<float, 32, false>(p, st);
  if (dt == SLA_F16) return p.phi == SLA_PHI_RELU ? fwd_launch<__half, 32, true>(p, st) : fwd_launch<__half, 32, false>(p, st);
  return p.phi == SLA_PHI_RELU ? fwd_launch<__nv_bfloat16, 32, true>(p, st) : fwd_launch<__nv_bfloat16, 32, false>(p, st);
}

cudaError_t launch_backward_generic(const Problem& p, int dt, cudaStream_t st) {
  if (p.d == 16) {
    if (dt == SLA_F32) return p.phi == SLA_PHI_RELU ? bwd_launch<float, 16, true>(p, st) : bwd_launch<float, 16, false>(p, st);
    if (dt == SLA_F16) return p.phi == SLA_PHI_RELU ? bwd_launch<__half, 16, true>(p, st) : bwd_launch<__half, 16, false>(p, st);
    return p.phi == SLA_PHI_RELU ? bwd_launch<__nv_bfloat16, 16, true>(p, st) : bwd_launch<__nv_bfloat16, 16, false>(p, st);
  }
  if (dt == SLA_F32) return p.phi == SLA_PHI_RELU ? bwd_launch<float, 32, true>(p, st) : bwd_launch<float, 32, false>(p, st);
  if (dt == SLA_F16) return p.phi == SLA_PHI_RELU ? bwd_launch<__half, 32, true>(p, st) : bwd_launch<__half, 32, false>(p, st);
  return p.phi == SLA_PHI_RELU ? bwd_launch<__nv_bfloat16, 32, true>(p, st) : bwd_launch<__nv_bfloat16, 32, false>(p, st);
}

}  // namespace sla
