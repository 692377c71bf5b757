// Probe: tcgen05.mma kind::f16, M=128, N=128, K=16 with BOTH operands MN-major straight from TMA tiles
// (row-major [rows x channels] fp16, box 64 cols x 16 rows, 128B swizzle).  D[r][p] = sum_j V[j][r]*K[j][p].
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
// MN-major (or K-major) shared-memory matrix descriptor, 128B swizzle, Blackwell version 1
__device__ __forceinline__ uint64_t make_desc(uint32_t addr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
  uint64_t d = 0;
  d |= (uint64_t)((addr >> 4) & 0x3FFF);
  d |= (uint64_t)((lbo_bytes >> 4) & 0x3FFF) << 16;
  d |= (uint64_t)((sbo_bytes >> 4) & 0x3FFF) << 32;
  d |= (uint64_t)1 << 46;    // version = 1
  d |= (uint64_t)2 << 61;    // SWIZZLE_128B
  return d;
}

constexpr int ROWS = 16, CH = 128;

__global__ void __launch_bounds__(128) probe(const __grid_constant__ CUtensorMap tmK, const __grid_constant__ CUtensorMap tmV,
                                              float* __restrict__ Dout, int lbo, int sbo) {
  extern __shared__ uint8_t dyn[];
  __shared__ unsigned long long bar_tma, bar_mma;
  __shared__ uint32_t tmem_base_s;
  const uint32_t base = (smem_u32(dyn) + 1023u) & ~1023u;
  const uint32_t Vs = base, Ks = base + 4096;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x == 0) {
    mbar_init(smem_u32(&bar_tma), 1);
    mbar_init(smem_u32(&bar_mma), 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_s)), "n"(128));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  asm volatile("tcgen05.fence::before_thread_sync;");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;");
  const uint32_t tmem = tmem_base_s;
  if (threadIdx.x == 0) {
    mbar_expect_tx(smem_u32(&bar_tma), 2 * 4096);
    tma_load_2d(Vs, &tmV, smem_u32(&bar_tma), 0, 0);
    tma_load_2d(Vs + 2048, &tmV, smem_u32(&bar_tma), 64, 0);
    tma_load_2d(Ks, &tmK, smem_u32(&bar_tma), 0, 0);
    tma_load_2d(Ks + 2048, &tmK, smem_u32(&bar_tma), 64, 0);
  }
  mbar_wait(smem_u32(&bar_tma), 0);
  asm volatile("tcgen05.fence::after_thread_sync;");
  if (threadIdx.x == 0) {
    const uint64_t da = make_desc(Vs, lbo, sbo), db = make_desc(Ks, lbo, sbo);
    // instruction descriptor: D=F32, A=B=F16, both MN-major, N=128, M=128
    const uint32_t idesc = (1u << 4) | (0u << 7) | (0u << 10) | (1u << 15) | (1u << 16) | ((128u >> 3) << 17) | ((128u >> 4) << 24);
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\ttcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}" ::"r"(tmem), "l"(da), "l"(db), "r"(idesc), "r"(0u) : "memory");
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(&bar_mma)) : "memory");
  }
  mbar_wait(smem_u32(&bar_mma), 0);
  asm volatile("tcgen05.fence::after_thread_sync;");
  // warp w reads TMEM lanes 32w .. 32w+31, 128 columns in chunks of 32
  for (int c = 0; c < 128; c += 32) {
    uint32_t r[32];
    const uint32_t taddr = tmem + ((uint32_t)(32 * warp) << 16) + (uint32_t)c;
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]),
          "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]), "=r"(r[17]), "=r"(r[18]),
          "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]),
          "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
        : "r"(taddr));
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
    for (int i = 0; i < 32; ++i) Dout[(size_t)(32 * warp + lane) * 128 + c + i] = __uint_as_float(r[i]);
  }
  asm volatile("tcgen05.fence::before_thread_sync;");
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(128));
}

int main(int argc, char** argv) {
  int lbo = argc > 1 ? atoi(argv[1]) : 2048, sbo = argc > 2 ? atoi(argv[2]) : 1024;
  std::vector<__half> hK(ROWS * CH), hV(ROWS * CH);
  srand(1);
  for (int i = 0; i < ROWS * CH; ++i) { hK[i] = __float2half((float)(rand() % 7 - 3)); hV[i] = __float2half((float)(rand() % 5 - 2)); }
  __half *dK, *dV; float* dD;
  cudaMalloc(&dK, ROWS * CH * 2); cudaMalloc(&dV, ROWS * CH * 2); cudaMalloc(&dD, 128 * 128 * 4);
  cudaMemcpy(dK, hK.data(), ROWS * CH * 2, cudaMemcpyHostToDevice);
  cudaMemcpy(dV, hV.data(), ROWS * CH * 2, cudaMemcpyHostToDevice);
  cudaMemset(dD, 0xff, 128 * 128 * 4);
  void* fp = nullptr; cudaDriverEntryPointQueryResult q;
  cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fp, cudaEnableDefault, &q);
  EncodeTiledFn enc = (EncodeTiledFn)fp;
  CUtensorMap tk, tv;
  const cuuint64_t dims[2] = {CH, ROWS}; const cuuint64_t strides[1] = {CH * 2};
  const cuuint32_t box[2] = {64, ROWS}; const cuuint32_t es[2] = {1, 1};
  CUresult r1 = enc(&tk, CU_TENSOR_MAP_DATA_TYPE_UINT16, 2, dK, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  CUresult r2 = enc(&tv, CU_TENSOR_MAP_DATA_TYPE_UINT16, 2, dV, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  printf("encode %d %d\n", (int)r1, (int)r2);
  cudaFuncSetAttribute(probe, cudaFuncAttributeMaxDynamicSharedMemorySize, 16384);
  probe<<<1, 128, 16384>>>(tk, tv, dD, lbo, sbo);
  cudaError_t e = cudaDeviceSynchronize();
  printf("kernel: %s\n", cudaGetErrorString(e));
  std::vector<float> hD(128 * 128);
  cudaMemcpy(hD.data(), dD, 128 * 128 * 4, cudaMemcpyDeviceToHost);
  double maxerr = 0, maxerrT = 0; int bad = 0;
  for (int r = 0; r < 128; ++r)
    for (int p = 0; p < 128; ++p) {
      float ref = 0, refT = 0;
      for (int j = 0; j < ROWS; ++j) {
        ref += __half2float(hV[j * CH + r]) * __half2float(hK[j * CH + p]);
        refT += __half2float(hV[j * CH + p]) * __half2float(hK[j * CH + r]);
      }
      double d = fabs(hD[r * 128 + p] - ref), dT = fabs(hD[r * 128 + p] - refT);
      if (d > maxerr) maxerr = d;
      if (dT > maxerrT) maxerrT = dT;
      if (d > 1e-3 && bad < 8) { printf("  D[%d][%d]=%g ref %g\n", r, p, hD[r * 128 + p], ref); ++bad; }
    }
  printf("lbo %d sbo %d: max err vs V^T K: %g ; vs K^T V: %g\n", lbo, sbo, maxerr, maxerrT);
  return 0;
}
