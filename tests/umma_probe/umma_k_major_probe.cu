// Probe 2: tcgen05.mma kind::f16, M=128, N=144, K=128 (8 k-steps) with K-major operands:
//   A = a TMA tile [128 rows x 128 channels] fp16 (two boxes of 64 channels, 128B swizzle), used in place;
//   B = [144 x 128] fp16 written by the threads with the 128B swizzle applied by hand.
//   O[i][n] = sum_k A[i][k] * B[n][k]
#include <cuda.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <cstdio>
#include <cstdlib>
#include <cstdint>
#include <vector>
#include <cmath>

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t c) { asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(c) : "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t b) { asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(b) : "memory"); }
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  uint32_t done;
  do {
    asm volatile("{\n\t.reg .pred P1;\n\tmbarrier.try_wait.parity.shared::cta.b64 P1, [%1], %2;\n\tselp.b32 %0, 1, 0, P1;\n\t}" : "=r"(done) : "r"(bar), "r"(parity) : "memory");
  } while (!done);
}
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* tm, uint32_t bar, int x, int y) {
  asm volatile("cp.async.bulk.tensor.2d.shared::cta.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];" ::"r"(dst), "l"(tm), "r"(bar), "r"(x), "r"(y) : "memory");
}
__device__ __forceinline__ uint64_t make_desc(uint32_t addr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
  uint64_t d = 0;
  d |= (uint64_t)((addr >> 4) & 0x3FFF);
  d |= (uint64_t)((lbo_bytes >> 4) & 0x3FFF) << 16;
  d |= (uint64_t)((sbo_bytes >> 4) & 0x3FFF) << 32;
  d |= (uint64_t)1 << 46;    // version = 1
  d |= (uint64_t)2 << 61;    // SWIZZLE_128B
  return d;
}
constexpr int M = 128, N = 144, KD = 128;
constexpr int A_BOX = M * 128, B_BOX = N * 128;   // bytes of one 64-channel box

__global__ void __launch_bounds__(128) probe2(const __grid_constant__ CUtensorMap tmA, const __half* __restrict__ Bg,
                                               float* __restrict__ Dout) {
  extern __shared__ uint8_t dyn[];
  __shared__ unsigned long long bar_tma, bar_mma;
  __shared__ uint32_t tmem_base_s;
  const uint32_t base = (smem_u32(dyn) + 1023u) & ~1023u;
  const uint32_t As = base, Bs = base + 2 * A_BOX;
  uint8_t* Bs_gen = dyn + (base - smem_u32(dyn)) + 2 * A_BOX;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x == 0) {
    mbar_init(smem_u32(&bar_tma), 1);
    mbar_init(smem_u32(&bar_mma), 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_s)), "n"(256));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  // B written by the threads: element (n, k) -> box k/64, row n, 16-byte chunk ((k%64)/8) ^ (n%8)
  for (int idx = threadIdx.x; idx < N * (KD / 8); idx += blockDim.x) {
    const int n = idx / (KD / 8), c = idx % (KD / 8);        // c: 16-byte chunk along k (8 elements)
    const int box = c >> 3, cib = c & 7;
    const uint4 v = *reinterpret_cast<const uint4*>(Bg + (size_t)n * KD + 8 * c);
    *reinterpret_cast<uint4*>(Bs_gen + box * B_BOX + n * 128 + ((cib ^ (n & 7)) << 4)) = v;
  }
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic writes -> visible to the tensor core proxy
  asm volatile("tcgen05.fence::before_thread_sync;");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;");
  const uint32_t tmem = tmem_base_s;
  if (threadIdx.x == 0) {
    mbar_expect_tx(smem_u32(&bar_tma), 2 * A_BOX);
    tma_load_2d(As, &tmA, smem_u32(&bar_tma), 0, 0);
    tma_load_2d(As + A_BOX, &tmA, smem_u32(&bar_tma), 64, 0);
  }
  mbar_wait(smem_u32(&bar_tma), 0);
  asm volatile("tcgen05.fence::after_thread_sync;");
  if (threadIdx.x == 0) {
    // D=F32, A=B=F16, both K-major, N=144, M=128
    const uint32_t idesc = (1u << 4) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
    for (int ks = 0; ks < KD / 16; ++ks) {
      const int box = ks >> 2, kin = ks & 3;                   // 4 k-steps of 16 elements (32 B) per 128-byte row
      const uint64_t da = make_desc(As + box * A_BOX + kin * 32, 16, 1024);
      const uint64_t db = make_desc(Bs + box * B_BOX + kin * 32, 16, 1024);
      asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\ttcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}" ::"r"(tmem), "l"(da), "l"(db), "r"(idesc), "r"(ks > 0 ? 1u : 0u) : "memory");
    }
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(&bar_mma)) : "memory");
  }
  mbar_wait(smem_u32(&bar_mma), 0);
  asm volatile("tcgen05.fence::after_thread_sync;");
  for (int c = 0; c < N; c += 16) {
    uint32_t r[16];
    const uint32_t taddr = tmem + ((uint32_t)(32 * warp) << 16) + (uint32_t)c;
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]),
          "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
        : "r"(taddr));
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
    for (int i = 0; i < 16; ++i) Dout[(size_t)(32 * warp + lane) * N + c + i] = __uint_as_float(r[i]);
  }
  asm volatile("tcgen05.fence::before_thread_sync;");
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(256));
}

int main() {
  std::vector<__half> hA(M * KD), hB(N * KD);
  srand(2);
  for (auto& x : hA) x = __float2half((float)(rand() % 7 - 3));
  for (auto& x : hB) x = __float2half((float)(rand() % 5 - 2));
  __half *dA, *dB; float* dD;
  cudaMalloc(&dA, M * KD * 2); cudaMalloc(&dB, N * KD * 2); cudaMalloc(&dD, M * N * 4);
  cudaMemcpy(dA, hA.data(), M * KD * 2, cudaMemcpyHostToDevice);
  cudaMemcpy(dB, hB.data(), N * KD * 2, cudaMemcpyHostToDevice);
  cudaMemset(dD, 0xff, M * N * 4);
  void* fp = nullptr; cudaDriverEntryPointQueryResult q;
  cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fp, cudaEnableDefault, &q);
  EncodeTiledFn enc = (EncodeTiledFn)fp;
  CUtensorMap ta;
  const cuuint64_t dims[2] = {KD, M}; const cuuint64_t strides[1] = {KD * 2};
  const cuuint32_t box[2] = {64, M}; const cuuint32_t es[2] = {1, 1};
  CUresult r1 = enc(&ta, CU_TENSOR_MAP_DATA_TYPE_UINT16, 2, dA, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  printf("encode %d\n", (int)r1);
  const int smem = 2 * A_BOX + 2 * B_BOX + 1024;
  cudaFuncSetAttribute(probe2, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
  probe2<<<1, 128, smem>>>(ta, dB, dD);
  cudaError_t e = cudaDeviceSynchronize();
  printf("kernel: %s\n", cudaGetErrorString(e));
  std::vector<float> hD(M * N);
  cudaMemcpy(hD.data(), dD, M * N * 4, cudaMemcpyDeviceToHost);
  double maxerr = 0; int bad = 0;
  for (int i = 0; i < M; ++i)
    for (int n = 0; n < N; ++n) {
      float ref = 0;
      for (int k = 0; k < KD; ++k) ref += __half2float(hA[i * KD + k]) * __half2float(hB[n * KD + k]);
      double d = fabs(hD[i * N + n] - ref);
      if (d > maxerr) maxerr = d;
      if (d > 1e-3 && bad < 8) { printf("  O[%d][%d]=%g ref %g\n", i, n, hD[i * N + n], ref); ++bad; }
    }
  printf("K-major M=128 N=144 K=128: max err %g\n", maxerr);
  return 0;
}
