// sla_tc_common.cuh -- helpers shared by the tensor-core kernels (forward and backward): PTX wrappers
// (mbarrier, TMA, ldmatrix, mma.sync), element/feature-map helpers, the per-warp ring view, the warp-wide
// window search and the host-side tensor-map encoder.
//
// Include it INSIDE the translation unit's `namespace sla { namespace { ... } }`, after defining
//   constexpr int NST  (ring stages per stream)  and  template <int D> struct Cfg { SR, BOX_BYTES, ... }.
#ifndef SLA_TC_COMMON_INCLUDED
#define SLA_TC_COMMON_INCLUDED

// ---- PTX wrappers ---------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  uint32_t done;
  do {
    asm volatile(
        "{\n\t.reg .pred P1;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%1], %2, %3;\n\t"
        "selp.b32 %0, 1, 0, P1;\n\t}"
        : "=r"(done) : "r"(bar), "r"(parity), "r"(20000u) : "memory");
  } while (!done);
}
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* tm, uint32_t bar, int x, int y) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cta.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
      ::"r"(dst), "l"(tm), "r"(bar), "r"(x), "r"(y) : "memory");
}
__device__ __forceinline__ void ldsm_x4(uint32_t addr, uint32_t (&r)[4]) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}
__device__ __forceinline__ void ldsm_x4_t(uint32_t addr, uint32_t (&r)[4]) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}
// D(16x8,f32) += A(16x16,f16,row) * B(16x8,f16,col)
__device__ __forceinline__ void mma16816(float (&c)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3,
                                         uint32_t b0, uint32_t b1) {
  asm(
      "mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
      : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
      : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}

// ---- element helpers ------------------------------------------------------------------------------
template <bool BF16>
__device__ __forceinline__ float2 unpack2(uint32_t r) {   // two packed I/O elements -> fp32
  if (BF16) return make_float2(__uint_as_float(r << 16), __uint_as_float(r & 0xffff0000u));
  return __half22float2(*reinterpret_cast<const __half2*>(&r));
}
__device__ __forceinline__ uint32_t pack_h2(float lo, float hi) {
  __half2 h = __floats2half2_rn(lo, hi);
  return *reinterpret_cast<uint32_t*>(&h);
}
template <bool BF16>
__device__ __forceinline__ uint32_t pack_out(float lo, float hi) {
  if (BF16) {
    __nv_bfloat162 b = __floats2bfloat162_rn(lo, hi);
    return *reinterpret_cast<uint32_t*>(&b);
  }
  return pack_h2(lo, hi);
}
// phi(x) = elu(x)+1 (reading A1); fast exp (ex2.approx) -- relative error ~2^-21, far below fp16 operands
// Branch-free: phi = max(x,0) + 2^min(x*log2e, 0)  (x > 0: x + 2^0 = x + 1 exactly; x <= 0: e^x), and the
// second term alone is phi'(x) = (x > 0 ? 1 : e^x).  One ex2.approx.ftz (relative error 2^-22) instead of
// __expf's range-checked sequence: 5 instructions per element.
__device__ __forceinline__ float ex2_fast(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float dphi_fast(float x) { return ex2_fast(fminf(x * 1.4426950408889634f, 0.f)); }
__device__ __forceinline__ float phi_fast(float x) { return fmaxf(x, 0.f) + dphi_fast(x); }

// phi on two packed I/O elements, evaluated in fp16x2 (long windows only: the operand is rounded to
// fp16 anyway).  Branch-free on the FMA pipe (the ALU pipe is the busy one in these kernels):
//   r = relu(x*log2e)            (fma.relu)
//   t = x*log2e - r = min(x*log2e, 0)   (one fused rounding)
//   phi = 2^t + r*ln2            x <= 0: r = 0, phi = 2^(x*log2e) = e^x
//                                x  > 0: t is only the rounding residual of r, 2^t = 1 + t*ln2 + ..., so
//                                        phi = 1 + x to first order in that residual (~1.5 fp16 ulp)
// Result: fp16x2 {phi(x0), phi(x1)}.
template <bool BF16>
__device__ __forceinline__ uint32_t phi_h2(uint32_t raw) {
  uint32_t x = raw;
  if (BF16) { float2 f = unpack2<true>(raw); x = pack_h2(f.x, f.y); }
  uint32_t r, t, e, out;
  const uint32_t log2e = 0x3DC53DC5u, ln2 = 0x398C398Cu, zero = 0u;   // fp16 1.4424, 0.6931
  asm("fma.rn.relu.f16x2 %0, %1, %2, %3;" : "=r"(r) : "r"(x), "r"(log2e), "r"(zero));
  asm("{\n\t.reg .b32 nr;\n\tneg.f16x2 nr, %3;\n\tfma.rn.f16x2 %0, %1, %2, nr;\n\t}"
      : "=r"(t) : "r"(x), "r"(log2e), "r"(r));
  asm("ex2.approx.f16x2 %0, %1;" : "=r"(e) : "r"(t));
  asm("fma.rn.f16x2 %0, %1, %2, %3;" : "=r"(out) : "r"(r), "r"(ln2), "r"(e));
  return out;
}
__device__ __forceinline__ float fast_rcp(float x) {
  float r;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}

// fp32 pair -> fp16x2 "hi" and the fp16x2 residual "lo"
__device__ __forceinline__ void split_h2(float x0, float x1, uint32_t& hi, uint32_t& lo) {
  __half2 h = __floats2half2_rn(x0, x1);
  float2 hf = __half22float2(h);
  hi = *reinterpret_cast<uint32_t*>(&h);
  lo = pack_h2(x0 - hf.x, x1 - hf.y);
}

// ---- per-warp consumer view of one ring -----------------------------------------------------------
// Stage st of a stream holds rows [R0 + st*SR, R0 + (st+1)*SR).  `waited` = stages whose full barrier
// this warp has observed; `released` = stages this warp has handed back to the producer.  The ring slot
// and barrier phase of the next stage to wait for / to release are tracked incrementally (no division
// by the stage count in the hot loops): stage st lives in slot (st + bias) mod NST for every stage that
// has not been released yet, with bias = r_slot - released.
struct RingView {
  uint32_t base;      // shared address of slot 0
  uint32_t full;      // shared address of full barriers [NST]
  uint32_t empty;     // shared address of empty barriers [NST]
  int waited;
  int released;
  int w_slot, w_phase;   // slot and parity of stage `waited`
  int r_slot, bias;      // slot of stage `released`; bias = r_slot - released
};
__device__ __forceinline__ RingView make_ring(uint32_t base, uint32_t full, uint32_t empty) {
  return RingView{base, full, empty, 0, 0, 0, 0, 0, 0};
}

__device__ __forceinline__ void ring_wait_upto(RingView& rv, int stage_last) {
  while (rv.waited <= stage_last) {
    mbar_wait(rv.full + 8u * rv.w_slot, (uint32_t)rv.w_phase);
    ++rv.waited;
    if (++rv.w_slot == NST) { rv.w_slot = 0; rv.w_phase ^= 1; }
  }
}
// Release every stage that lies entirely below relative row `rel` (rows are relative to R0).
template <int SR>
__device__ __forceinline__ void ring_release_below(RingView& rv, int rel) {
  while ((rv.released + 1) * SR <= rel) {
    ring_wait_upto(rv, rv.released);   // never release a stage before it has landed (phase pacing)
    __syncwarp();
    if ((threadIdx.x & 31) == 0) mbar_arrive(rv.empty + 8u * rv.r_slot);
    ++rv.released;
    if (++rv.r_slot == NST) { rv.r_slot = 0; rv.bias -= NST; }
  }
}
// Steady state of a loop whose step is exactly one stage of rows: after the first step of a pass,
// every further step starts SR rows later, so exactly one more stage -- the oldest unreleased one, which
// the previous step has read and therefore waited for -- lies entirely below it.
__device__ __forceinline__ void ring_release_one(RingView& rv) {
  __syncwarp();
  if ((threadIdx.x & 31) == 0) mbar_arrive(rv.empty + 8u * rv.r_slot);
  ++rv.released;
  if (++rv.r_slot == NST) { rv.r_slot = 0; rv.bias -= NST; }
}

// Shared address of (relative row rel, 16-byte chunk `chunk` of this slab row) inside a ring whose
// slots are `slot_bytes` apart; the tensor's stage starts `toff` bytes into the slot.  The row must
// belong to a stage that has been waited for and not yet released.
template <int D>
__device__ __forceinline__ uint32_t ring_addr(const RingView& rv, int slot_bytes, int toff, int rel, int chunk) {
  using C = Cfg<D>;
  const int st = (int)((unsigned)rel / (unsigned)C::SR), r = (int)((unsigned)rel % (unsigned)C::SR);   // rel >= 0
  int slot = st + rv.bias;
  if (slot >= NST) slot -= NST;
  const int box = chunk >> 3, cib = chunk & 7;
  return rv.base + (uint32_t)(slot * slot_bytes + toff + box * C::BOX_BYTES + r * 128 +
                              ((cib ^ (r & 7)) << 4));
}

// For two rows at once (independent probes in flight together): the largest w in [0,W) with
// off[w] <= row (row < off[W] = N), found by one warp with 32-way probes per round.
__device__ __forceinline__ void warp_windows_of_rows(const int32_t* __restrict__ off, int W, int rowa,
                                                     int rowb, int& wa, int& wb) {
  const int lane = threadIdx.x & 31;
  int lo[2] = {0, 0}, hi[2] = {W, W};
  const int row[2] = {rowa, rowb};
  while (hi[0] - lo[0] > 1 || hi[1] - lo[1] > 1) {
    int step[2], idx[2], val[2];
#pragma unroll
    for (int k = 0; k < 2; ++k) {
      step[k] = max(1, (hi[k] - lo[k] + 31) / 32);
      idx[k] = lo[k] + (lane + 1) * step[k];
      val[k] = __ldg(off + min(idx[k], W));
    }
#pragma unroll
    for (int k = 0; k < 2; ++k) {
      const bool ok = idx[k] < hi[k] && val[k] <= row[k];
      const int cnt = __popc(__ballot_sync(0xffffffffu, ok));
      const int nlo = lo[k] + cnt * step[k];
      hi[k] = min(hi[k], nlo + step[k]);
      lo[k] = nlo;
    }
  }
  wa = lo[0];
  wb = lo[1];
}

// ---- host side -------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*,
                                  CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                  CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn() {
  static EncodeTiledFn fn = []() -> EncodeTiledFn {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess ||
        q != cudaDriverEntryPointSuccess)
      return nullptr;
    return reinterpret_cast<EncodeTiledFn>(p);
  }();
  return fn;
}

// 2-D map over a row-major [N, C] 16-bit tensor; box = 64 columns (128 B) x box_rows, 128-B swizzle.
bool make_map(CUtensorMap* tm, const void* base, int N, int C, int box_rows) {
  EncodeTiledFn enc = encode_fn();
  if (!enc) return false;
  const cuuint64_t dims[2] = {(cuuint64_t)C, (cuuint64_t)N};
  const cuuint64_t strides[1] = {(cuuint64_t)C * 2};
  const cuuint32_t box[2] = {64u, (cuuint32_t)box_rows};
  const cuuint32_t estr[2] = {1u, 1u};
  return enc(tm, CU_TENSOR_MAP_DATA_TYPE_UINT16, 2, const_cast<void*>(base), dims, strides, box, estr,
             CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// Per-device caches (a process may drive several GPUs): index = current CUDA device.
constexpr int kMaxDevices = 64;
int current_device() {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) dev = 0;
  return dev;
}
int sm_count() {
  static std::atomic<int> cache[kMaxDevices];
  const int dev = current_device();
  int v = cache[dev].load(std::memory_order_relaxed);
  if (v <= 0) {
    v = 148;
    cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev);
    if (v <= 0) v = 148;
    cache[dev].store(v, std::memory_order_relaxed);
  }
  return v;
}

#endif  // SLA_TC_COMMON_INCLUDED
