// sla_proj.cu -- the shared Q/K/V projection around the SLA op: Q = x W_Q, K = x W_K, V = x W_V
// (PAPER.md:71, 77), one GEMM  y[N, 3C] = x[N, C] . w[3C, C]^T (+ bias)  on the 5th-generation tensor cores.
//
// A dense contraction, so it goes to tcgen05: one persistent CTA per SM walks 128-row tiles of x.
//   warp 0 (one lane)   producer: TMA loads of the x tile (128 x C, K-major, 128-byte swizzle) and, per chunk of 128
//                       output features, of the matching 128 rows of w (also K-major: w is [out, in]); w comes out of L2
//   warp 1 (one lane)   issues tcgen05.mma M=128 N=128 K=16, C/16 of them per chunk, accumulating in tensor memory
//                       (two 128-column accumulators: chunk j+1 is multiplied while chunk j is drained)
//   warps 2-5           epilogue: tcgen05.ld (one row of the tile per thread), + bias, round to the I/O dtype, stage the
//                       128 x 128 block in shared memory in the swizzled box layout, one TMA store per 64-column box into
//                       q, k or v (chunk j covers output features 128 j ..: tensor (128 j) / C, column (128 j) % C);
//                       rows beyond N are clipped by the TMA unit
// HBM-bound: 2 N C 3C flops on N C + 3 N C elements moved (47 flop/B at C = 128, a tenth of the machine balance).
#include <cuda.h>

#include <atomic>

#include "sla_internal.cuh"

namespace sla {
namespace {

#include "sla_tc_base.cuh"

constexpr int TILE_M = 128;      // rows of x per tile = TMEM lanes
constexpr int CHUNK_N = 128;     // output features per accumulator
constexpr int BOX_BYTES = TILE_M * 128;   // one 64-column box of a 128-row tile (16 KB)
constexpr int TMEM_COLS = 2 * CHUNK_N;
constexpr int WARP_PRODUCER = 0, WARP_MMA = 1, WARP_EPI0 = 2, NUM_EPI_WARPS = 4;
constexpr int THREADS = (WARP_EPI0 + NUM_EPI_WARPS) * 32;

template <int C> struct Cfg {
  static constexpr int KB = C / 64;                       // 64-column boxes along K
  static constexpr int KSTEPS = C / 16;
  static constexpr int OPERAND_BYTES = KB * BOX_BYTES;    // a 128 x C operand tile
  static constexpr int NA = (C <= 128) ? 2 : 1;           // x-tile stages
  static constexpr int NWS = 2;                           // w-chunk stages
  static constexpr int NOS = (C <= 128) ? 2 : 1;          // output staging buffers (128 x 128 elements, 32 KB)
  static constexpr int OFF_A = 0;
  static constexpr int OFF_W = OFF_A + NA * OPERAND_BYTES;
  static constexpr int OFF_O = OFF_W + NWS * OPERAND_BYTES;
  static constexpr int SMEM_DYN = OFF_O + NOS * 2 * BOX_BYTES + 1024;   // + alignment slack (swizzle needs 1 KB)
};

struct Ctrl {
  unsigned long long a_full[2], a_empty[2], w_full[2], w_empty[2], acc_full[2], acc_empty[2];
  uint32_t tmem_base;
};

struct Maps { CUtensorMap x, w, out[3]; };

// ---- tcgen05 / TMA-store wrappers ---------------------------------------------------------------------
// shared-memory matrix descriptor, K-major operand in 64-column boxes, 128-byte swizzle, descriptor version 1:
// start address, leading byte offset (unused for swizzled K-major: 16), stride byte offset = 8 rows x 128 B
__device__ __forceinline__ uint64_t make_desc(uint32_t addr) {
  uint64_t d = 0;
  d |= (uint64_t)((addr >> 4) & 0x3FFF);
  d |= (uint64_t)(16u >> 4) << 16;
  d |= (uint64_t)(1024u >> 4) << 32;
  d |= (uint64_t)1 << 46;
  d |= (uint64_t)2 << 61;
  return d;
}
// instruction descriptor of kind::f16: fp32 accumulate, both operands K-major, formats fp16 (0) or bf16 (1)
__host__ __device__ constexpr uint32_t make_idesc(int M, int N, bool bf16) {
  return (1u << 4) | ((bf16 ? 1u : 0u) << 7) | ((bf16 ? 1u : 0u) << 10) | ((uint32_t)(N >> 3) << 17) |
         ((uint32_t)(M >> 4) << 24);
}
__device__ __forceinline__ void umma(uint32_t d_tmem, uint64_t a, uint64_t b, uint32_t idesc, uint32_t acc) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
      ::"r"(d_tmem), "l"(a), "l"(b), "r"(idesc), "r"(acc) : "memory");
}
__device__ __forceinline__ void umma_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&r)[32]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,"
      "%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
        "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]),
        "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]),
        "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
      : "r"(taddr));
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void sts128(uint32_t a, uint32_t x, uint32_t y, uint32_t z, uint32_t w) {
  asm volatile("st.shared.v4.u32 [%0], {%1,%2,%3,%4};" ::"r"(a), "r"(x), "r"(y), "r"(z), "r"(w) : "memory");
}
__device__ __forceinline__ void tma_store_2d(const CUtensorMap* tm, uint32_t src, int x, int y) {
  asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%2, %3}], [%1];"
               ::"l"(tm), "r"(src), "r"(x), "r"(y) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int PENDING>
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(PENDING) : "memory"); }
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
// mbarrier wait with a watchdog: a protocol error traps instead of hanging the device
__device__ __forceinline__ void mbar_wait_wd(uint32_t bar, uint32_t parity) {
  uint32_t done, spins = 0;
  do {
    asm volatile(
        "{\n\t.reg .pred P1;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%1], %2, %3;\n\t"
        "selp.b32 %0, 1, 0, P1;\n\t}"
        : "=r"(done) : "r"(bar), "r"(parity), "r"(100000u) : "memory");
    if (!done && ++spins > (1u << 16)) __trap();
  } while (!done);
}
// a ring cursor: stage index and the parity of its next completion
struct Cur { int s; uint32_t ph; };
template <int N> __device__ __forceinline__ void advance(Cur& c) { if (++c.s == N) { c.s = 0; c.ph ^= 1u; } }

template <int C, bool BF16, typename T>
__global__ void __launch_bounds__(THREADS, 1)
sla_qkv_proj_kernel(const __grid_constant__ Maps maps, const float* __restrict__ bias, int N, int nch) {
  // nch = chunks of 128 output features = (number of [N, C] output tensors: 3 for q, k, v; 1 for a plain layer) * C / 128
  using G = Cfg<C>;
  extern __shared__ uint8_t dyn_smem[];
  __shared__ Ctrl ctrl;
  asm volatile("griddepcontrol.launch_dependents;");
  const uint32_t sbase = (smem_u32(dyn_smem) + 1023u) & ~1023u;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  // Work unit = (128-row tile, 128-feature chunk).  Every CTA takes one contiguous range of units, so the ranges differ
  // by at most one chunk (a third of a tile at C = 128) where whole tiles would differ by one tile in ~3; a tile that
  // straddles two ranges is loaded by both CTAs (the second time out of L2).
  const long long units = (long long)((N + TILE_M - 1) / TILE_M) * nch;
  const int u0 = (int)(units * blockIdx.x / gridDim.x), u1 = (int)(units * (blockIdx.x + 1) / gridDim.x);

  if (threadIdx.x == 0) {
    for (int i = 0; i < 2; ++i) {
      mbar_init(smem_u32(&ctrl.a_full[i]), 1);
      mbar_init(smem_u32(&ctrl.a_empty[i]), 1);
      mbar_init(smem_u32(&ctrl.w_full[i]), 1);
      mbar_init(smem_u32(&ctrl.w_empty[i]), 1);
      mbar_init(smem_u32(&ctrl.acc_full[i]), 1);
      mbar_init(smem_u32(&ctrl.acc_empty[i]), NUM_EPI_WARPS);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == WARP_MMA) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;"
                 ::"r"(smem_u32(&ctrl.tmem_base)), "n"(TMEM_COLS));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  // nothing the previous kernel of the stream may have written (x, w, bias) or may still read (q, k, v) is touched
  // before this returns
  asm volatile("griddepcontrol.wait;" ::: "memory");
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = ctrl.tmem_base;

  if (warp == WARP_PRODUCER) {
    if (lane == 0) {
      Cur a{0, 0}, w{0, 0};
      for (int u = u0; u < u1; ++u) {
        const int tile = u / nch, j = u % nch;
        if (j == 0 || u == u0) {                                     // first unit of a tile in this range: its x rows
          mbar_wait_wd(smem_u32(&ctrl.a_empty[a.s]), a.ph ^ 1u);     // passes at once on a stage never used
          const uint32_t abar = smem_u32(&ctrl.a_full[a.s]);
          mbar_expect_tx(abar, (uint32_t)G::OPERAND_BYTES);
#pragma unroll
          for (int b = 0; b < G::KB; ++b)
            tma_load_2d(sbase + G::OFF_A + a.s * G::OPERAND_BYTES + b * BOX_BYTES, &maps.x, abar, 64 * b, tile * TILE_M);
          advance<G::NA>(a);
        }
        mbar_wait_wd(smem_u32(&ctrl.w_empty[w.s]), w.ph ^ 1u);
        const uint32_t wbar = smem_u32(&ctrl.w_full[w.s]);
        mbar_expect_tx(wbar, (uint32_t)G::OPERAND_BYTES);
#pragma unroll
        for (int b = 0; b < G::KB; ++b)
          tma_load_2d(sbase + G::OFF_W + w.s * G::OPERAND_BYTES + b * BOX_BYTES, &maps.w, wbar, 64 * b, CHUNK_N * j);
        advance<G::NWS>(w);
      }
    }
  } else if (warp == WARP_MMA) {
    if (lane == 0) {
      constexpr uint32_t IDESC = make_idesc(TILE_M, CHUNK_N, BF16);
      Cur a{0, 0}, w{0, 0}, acc{0, 0};
      for (int u = u0; u < u1; ++u) {
        const int j = u % nch;
        if (j == 0 || u == u0) mbar_wait_wd(smem_u32(&ctrl.a_full[a.s]), a.ph);
        const uint32_t abase = sbase + G::OFF_A + a.s * G::OPERAND_BYTES;
        mbar_wait_wd(smem_u32(&ctrl.w_full[w.s]), w.ph);
        mbar_wait_wd(smem_u32(&ctrl.acc_empty[acc.s]), acc.ph ^ 1u);
        tc_fence_after();
        const uint32_t wbase = sbase + G::OFF_W + w.s * G::OPERAND_BYTES;
#pragma unroll
        for (int ks = 0; ks < G::KSTEPS; ++ks) {
          // k-step ks = 16 columns = 32 bytes inside the 128-byte row of box ks/4
          const uint32_t koff = (uint32_t)((ks >> 2) * BOX_BYTES + (ks & 3) * 32);
          umma(tmem + (uint32_t)(acc.s * CHUNK_N), make_desc(abase + koff), make_desc(wbase + koff), IDESC,
               ks > 0 ? 1u : 0u);
        }
        umma_commit(smem_u32(&ctrl.w_empty[w.s]));       // the w stage may be overwritten once these MMAs have read it
        umma_commit(smem_u32(&ctrl.acc_full[acc.s]));
        advance<G::NWS>(w);
        advance<2>(acc);
        if (j == nch - 1 || u == u1 - 1) {             // last unit of the tile in this range: hand the x stage back
          umma_commit(smem_u32(&ctrl.a_empty[a.s]));
          advance<G::NA>(a);
        }
      }
    }
  } else {
    // ---- epilogue: thread = one row of the tile (TMEM lane 32 (warp % 4) + lane) ----
    const int q4 = warp & 3;
    const int row = 32 * q4 + lane;
    const int et = threadIdx.x - WARP_EPI0 * 32;            // 0..127
    Cur acc{0, 0};
    int os = 0;                                              // staging buffer of the next chunk
    {
      for (int u = u0; u < u1; ++u) {
        const int tile = u / nch, j = u % nch;
        // the staging buffer must have been read by the bulk store of the chunk that used it last
        if (et == 0) bulk_wait_read<G::NOS - 1>();
        asm volatile("bar.sync 1, 128;" ::: "memory");
        mbar_wait_wd(smem_u32(&ctrl.acc_full[acc.s]), acc.ph);
        tc_fence_after();
        const uint32_t obuf = sbase + G::OFF_O + os * 2 * BOX_BYTES;
#pragma unroll
        for (int p = 0; p < CHUNK_N / 32; ++p) {
          uint32_t r[32];
          tmem_ld32(tmem + ((uint32_t)(32 * q4) << 16) + (uint32_t)(acc.s * CHUNK_N + 32 * p), r);
          uint32_t h[16];
          if (bias != nullptr) {                               // the same 32 values for every thread: broadcast loads
            const float4* bp = reinterpret_cast<const float4*>(bias + CHUNK_N * j + 32 * p);
#pragma unroll
            for (int i = 0; i < 8; ++i) {
              const float4 b = __ldg(bp + i);
              h[2 * i] = pack_out<BF16>(__uint_as_float(r[4 * i]) + b.x, __uint_as_float(r[4 * i + 1]) + b.y);
              h[2 * i + 1] = pack_out<BF16>(__uint_as_float(r[4 * i + 2]) + b.z, __uint_as_float(r[4 * i + 3]) + b.w);
            }
          } else {
#pragma unroll
            for (int i = 0; i < 16; ++i) h[i] = pack_out<BF16>(__uint_as_float(r[2 * i]), __uint_as_float(r[2 * i + 1]));
          }
          // columns 32 p .. 32 p + 31 = box p/2, 16-byte chunks 4 (p%2) .. 4 (p%2) + 3 of this row's 128 bytes
          const uint32_t rbase = obuf + (uint32_t)((p >> 1) * BOX_BYTES + row * 128);
#pragma unroll
          for (int c4 = 0; c4 < 4; ++c4) {
            const int c = 4 * (p & 1) + c4;
            sts128(rbase + (uint32_t)(((c ^ (row & 7)) << 4)), h[4 * c4], h[4 * c4 + 1], h[4 * c4 + 2], h[4 * c4 + 3]);
          }
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(smem_u32(&ctrl.acc_empty[acc.s]));
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic-proxy writes -> visible to the TMA unit
        asm volatile("bar.sync 1, 128;" ::: "memory");
        if (et == 0) {
          const int f0 = CHUNK_N * j;                                  // first output feature of the chunk
          const CUtensorMap* tm = &maps.out[f0 / C];
          tma_store_2d(tm, obuf, f0 % C, tile * TILE_M);
          tma_store_2d(tm, obuf + BOX_BYTES, f0 % C + 64, tile * TILE_M);
          bulk_commit();
        }
        advance<2>(acc);
        if (++os == G::NOS) os = 0;
      }
    }
    if (et == 0) bulk_wait_all();
  }
  tc_fence_before();
  __syncthreads();
  if (warp == WARP_MMA) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(TMEM_COLS));
  }
}

// n_out = 3: w is [3C, C], outputs q, k, v; n_out = 1: w is [C, C], one output (k and v unused)
template <int C, bool BF16, typename T>
cudaError_t proj_launch(const void* x, const void* w, const float* bias, int N, int n_out, void* q, void* k, void* v,
                        cudaStream_t st) {
  using G = Cfg<C>;
  Maps maps;
  if (!make_map(&maps.x, x, N, C, TILE_M) || !make_map(&maps.w, w, n_out * C, C, CHUNK_N) ||
      !make_map(&maps.out[0], q, N, C, TILE_M))
    return cudaErrorInvalidValue;
  maps.out[1] = maps.out[0];
  maps.out[2] = maps.out[0];
  if (n_out == 3 && (!make_map(&maps.out[1], k, N, C, TILE_M) || !make_map(&maps.out[2], v, N, C, TILE_M)))
    return cudaErrorInvalidValue;
  auto kern = sla_qkv_proj_kernel<C, BF16, T>;
  static std::atomic<bool> attr_set[kMaxDevices];         // the smem opt-in is per device
  const int dev = current_device();
  if (!attr_set[dev].load(std::memory_order_acquire)) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, G::SMEM_DYN);
    if (e != cudaSuccess) return e;
    attr_set[dev].store(true, std::memory_order_release);
  }
  const int ntiles = (N + TILE_M - 1) / TILE_M;
  cudaLaunchAttribute pdl[1];
  pdl[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  pdl[0].val.programmaticStreamSerializationAllowed = 1;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(ntiles < sm_count() ? ntiles : sm_count());   // persistent: one CTA per SM
  cfg.blockDim = dim3(THREADS);
  cfg.dynamicSmemBytes = G::SMEM_DYN;
  cfg.stream = st;
  cfg.attrs = pdl;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kern, maps, bias, N, n_out * C / CHUNK_N);
}

// ---- generic path: fp32 I/O and every C the tensor-core kernel does not take ------------------------------------------
// A plain shared-memory tiled product on the CUDA cores, fp32 accumulation in a fixed order: 64 rows x 64 output
// features per block, 16 columns of x and w per step, 4 x 4 outputs per thread.  A fallback, not a fast path.
template <typename T> __device__ __forceinline__ float to_f32(T v);
template <> __device__ __forceinline__ float to_f32<float>(float v) { return v; }
template <> __device__ __forceinline__ float to_f32<__half>(__half v) { return __half2float(v); }
template <> __device__ __forceinline__ float to_f32<__nv_bfloat16>(__nv_bfloat16 v) { return __bfloat162float(v); }
template <typename T> __device__ __forceinline__ T from_f32(float v);
template <> __device__ __forceinline__ float from_f32<float>(float v) { return v; }
template <> __device__ __forceinline__ __half from_f32<__half>(float v) { return __float2half_rn(v); }
template <> __device__ __forceinline__ __nv_bfloat16 from_f32<__nv_bfloat16>(float v) { return __float2bfloat16_rn(v); }

constexpr int GT = 64, GK = 16;

template <typename T>
__global__ void __launch_bounds__(256)
sla_proj_generic_kernel(const T* __restrict__ x, const T* __restrict__ w, const float* __restrict__ bias, int N, int C,
                        int F /* output features = n_out * C */, T* __restrict__ y0, T* __restrict__ y1,
                        T* __restrict__ y2) {
  __shared__ float sx[GK][GT + 1], sw[GK][GT + 1];
  asm volatile("griddepcontrol.launch_dependents;");
  asm volatile("griddepcontrol.wait;" ::: "memory");
  const int row0 = blockIdx.x * GT, f0 = blockIdx.y * GT;
  const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;      // thread: rows 4 ty .., features 4 tx ..
  float acc[4][4] = {};
  for (int k0 = 0; k0 < C; k0 += GK) {
    for (int i = threadIdx.x; i < GT * GK; i += 256) {
      const int r = i / GK, kk = i % GK;
      const bool kin = k0 + kk < C;
      sx[kk][r] = (kin && row0 + r < N) ? to_f32<T>(x[(size_t)(row0 + r) * C + k0 + kk]) : 0.f;
      sw[kk][r] = (kin && f0 + r < F) ? to_f32<T>(w[(size_t)(f0 + r) * C + k0 + kk]) : 0.f;
    }
    __syncthreads();
#pragma unroll
    for (int kk = 0; kk < GK; ++kk) {
      float a[4], b[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) { a[i] = sx[kk][4 * ty + i]; b[i] = sw[kk][4 * tx + i]; }
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(a[i], b[j], acc[i][j]);
    }
    __syncthreads();
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int r = row0 + 4 * ty + i;
    if (r >= N) continue;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int f = f0 + 4 * tx + j;
      if (f >= F) continue;
      const float v = acc[i][j] + (bias != nullptr ? __ldg(bias + f) : 0.f);
      T* y = (f < C) ? y0 : (f < 2 * C ? y1 : y2);             // feature block -> output tensor
      y[(size_t)r * C + (f % C)] = from_f32<T>(v);
    }
  }
}

template <typename T>
cudaError_t proj_generic_launch(const void* x, const void* w, const float* bias, int N, int C, int n_out, void* q,
                                void* k, void* v, cudaStream_t st) {
  cudaLaunchAttribute pdl[1];
  pdl[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  pdl[0].val.programmaticStreamSerializationAllowed = 1;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((N + GT - 1) / GT, (n_out * C + GT - 1) / GT);
  cfg.blockDim = dim3(256);
  cfg.stream = st;
  cfg.attrs = pdl;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, sla_proj_generic_kernel<T>, (const T*)x, (const T*)w, bias, N, C, n_out * C, (T*)q,
                            (T*)k, (T*)v);
}

}  // namespace

// the tcgen05 kernel takes fp16 / bf16 with C = 128 or 256; everything else (fp32 I/O, other C) the generic kernel
static bool projection_on_tensor_cores(int C, int dt) {
  return (dt == SLA_F16 || dt == SLA_BF16) && (C == 128 || C == 256) && encode_fn() != nullptr;
}

bool qkv_projection_supported(int C, int dt) {
  return (dt == SLA_F32 || dt == SLA_F16 || dt == SLA_BF16) && C >= 1 && C <= (1 << 20);
}

cudaError_t launch_qkv_projection(const void* x, const void* w, const float* bias, int N, int C, int dt, int n_out,
                                  void* q, void* k, void* v, cudaStream_t st) {
  if (!projection_on_tensor_cores(C, dt)) {
    if (dt == SLA_F32) return proj_generic_launch<float>(x, w, bias, N, C, n_out, q, k, v, st);
    if (dt == SLA_F16) return proj_generic_launch<__half>(x, w, bias, N, C, n_out, q, k, v, st);
    return proj_generic_launch<__nv_bfloat16>(x, w, bias, N, C, n_out, q, k, v, st);
  }
  if (C == 128)
    return dt == SLA_F16 ? proj_launch<128, false, __half>(x, w, bias, N, n_out, q, k, v, st)
                         : proj_launch<128, true, __nv_bfloat16>(x, w, bias, N, n_out, q, k, v, st);
  return dt == SLA_F16 ? proj_launch<256, false, __half>(x, w, bias, N, n_out, q, k, v, st)
                       : proj_launch<256, true, __nv_bfloat16>(x, w, bias, N, n_out, q, k, v, st);
}

}  // namespace sla
