// sla_fwd_umma.cu -- SLA forward on the 5th-generation tensor cores (tcgen05.mma, accumulators in TMEM), all heads
// of a 128-channel slab at once.  fp16 / bf16 I/O, d_h = 16, H*d_h a multiple of 128.
//
// What is computed (Eq. 2-3): per window w and head h
//     S = sum_j phi(k_j)^T v_j,   z = sum_j phi(k_j),   o_i = phi(q_i) S / (phi(q_i) . z).
//
// Design:
//   * One persistent CTA per SM; the flat window-sorted matrix is cut into one row span per CTA
//     (load balance by rows, Fig. 3a).  A CTA owns every window of <= kFuseMax rows whose middle
//     row lies in its span, and the pieces of longer windows that intersect it (partial state -> fp32 atomics
//     into the workspace; their outputs come from the OUTPASS launch of sla_fwd_tc.cu).
//   * A producer warp walks the window offsets and turns them into ITEMS (a descriptor ring in shared memory):
//       PACK   consecutive whole windows of <= 16 rows, together <= 16 rows: one packed tile, masked quadratic
//              form on mma.sync with split operands (quad_tile_core) -- the fp16-operand linear form does not
//              meet the tolerance on windows this short;
//       WIN    one window of 17..kFuseMax rows;
//       PIECE  the part of a longer window inside this span (state only).
//     For every item it issues 2-D TMA loads (box 64 channels x 16 rows, 128-byte swizzle) of exactly that
//     item's rows: K,V tiles of 16 rows into a ring, Q blocks of up to 128 rows into block buffers.
//   * K-group warps apply phi to each K tile IN PLACE (rows past the window end are zeroed: the contraction of
//     the state MMA runs over rows); the MMA warp then issues, per 16 rows,
//         D[r][p]  += sum_j V[j][r] phi(K)[j][p]      tcgen05.mma M=128 N=128 K=16, both operands MN-major,
//         Z[p][.]  += sum_j phi(K)[j][p] * 1          tcgen05.mma M=128 N=16  K=16 against a tile of ones,
//     straight from the TMA tiles.  The 16x16 diagonal blocks of D are the per-head states S_h^T; the
//     off-diagonal blocks (7/8 of the tensor work, ~64 cycles per 16 rows) are ignored.
//   * When a window's state is complete the K-group reads its diagonal blocks and z from TMEM, scales them by
//     2^-ceil(log2 m) (Eq. 3 is a ratio) and writes them as fp16 B operands: per head a [16 x 16] K-major tile
//     (row r = S_h[.][r]) and one [8 x 128] tile of the z_h.
//   * Q-group warps apply phi to the Q block in place; the MMA warp issues per head
//         O[i][16h..16h+15] = phi(Q)[i][16h..16h+15] . B_h^T    M=128 N=16 K=16
//     and the denominators  O[i][128+h] = phi(Q)[i][:] . Bden[h][:]   M=128 N=16 K=128,
//     into the TMEM columns the state occupied; the Q-group reads its rows back (one thread per row), divides and
//     stores 32 contiguous bytes per head with 128-bit stores.
//   * Precision: operands fp16 (bf16 inputs: V is consumed as bf16 by the tensor core, K and Q are converted
//     when phi is applied), accumulation fp32.
#include <cuda.h>

#include <atomic>

#include "sla_internal.cuh"

namespace sla {
namespace {

#include "sla_tc_base.cuh"

constexpr int D = 16;                       // head dim of this kernel
constexpr int HS = 128 / D;                 // heads per 128-channel slab
constexpr int NKV = 6;                      // K/V tile ring: slots of [K 16x128 | V 16x128] fp16 = 8 KB
constexpr int NQB = 3;                      // Q block buffers: [128 rows x 128 ch] fp16 = 32 KB
constexpr int NSL = 3;                      // TMEM regions of 144 columns (state, then output, of one item)
constexpr int NB = 2;                       // B operand buffers (8 head tiles of 2 KB + 4 KB of z)
constexpr int NPK = 2;                      // packed-tile slots [K | V | Q] 16 rows each = 12 KB
constexpr int NIT = 8;                      // item descriptor ring
constexpr int KG_WARPS = 8, QG_WARPS = 8;
constexpr int WARP_PROD = 0, WARP_MMA = 1, WARP_KG0 = 2, WARP_QG0 = WARP_KG0 + KG_WARPS;
constexpr int THREADS = (2 + KG_WARPS + QG_WARPS) * 32;
constexpr int TILE_BYTES = 4096;            // 16 rows x 128 channels fp16 (two 64-channel boxes of 2 KB)
constexpr int KV_SLOT = 2 * TILE_BYTES, Q_BUF = 8 * TILE_BYTES, PK_SLOT = 3 * TILE_BYTES;
constexpr int BH_BYTES = 2048, B_BUF = HS * BH_BYTES + 4096, ONES_BYTES = 2048;
constexpr int OFF_KV = 0, OFF_Q = OFF_KV + NKV * KV_SLOT, OFF_B = OFF_Q + NQB * Q_BUF,
              OFF_PK = OFF_B + NB * B_BUF, OFF_ONES = OFF_PK + NPK * PK_SLOT;
constexpr int SMEM_DYN = OFF_ONES + ONES_BYTES + 1024;      // + alignment slack (swizzle needs 1 KB)
constexpr int REGION_COLS = 144, TMEM_COLS = 512;
constexpr int PF_AHEAD = 512, PF_CHUNK = 64;                // L2 prefetch distance / granularity in rows

enum ItemType { IT_END = 0, IT_PACK = 1, IT_WIN = 2, IT_PIECE = 3 };

struct Ctrl {
  unsigned long long item_full[NIT], item_empty[NIT];
  unsigned long long kv_full[NKV], kphi[NKV], kv_empty[NKV];
  unsigned long long q_full[NQB], qphi[NQB], q_empty[NQB];
  unsigned long long state_full[NSL], region_free[NSL], o_full[NSL], o_drained[NSL];
  unsigned long long b_full[NB], b_empty[NB];
  unsigned long long pk_full[NPK], pk_empty[NPK];
  int4 items[NIT];
  uint32_t tmem_base;
};

// ring cursor: slot index and the parity of the current use of that slot
struct Cur {
  int slot;
  uint32_t phase;
};
template <int N>
__device__ __forceinline__ void advance(Cur& c) {
  if (++c.slot == N) { c.slot = 0; c.phase ^= 1u; }
}

// ---- tcgen05 wrappers --------------------------------------------------------------------------------
// shared-memory matrix descriptor, 128-byte swizzle, Blackwell descriptor version 1
__device__ __forceinline__ uint64_t make_desc(uint32_t addr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
  uint64_t d = 0;
  d |= (uint64_t)((addr >> 4) & 0x3FFF);
  d |= (uint64_t)((lbo_bytes >> 4) & 0x3FFF) << 16;
  d |= (uint64_t)((sbo_bytes >> 4) & 0x3FFF) << 32;
  d |= (uint64_t)1 << 46;
  d |= (uint64_t)2 << 61;
  return d;
}
// instruction descriptor of kind::f16: fp32 accumulate; a_bf16 / b_bf16 select the operand formats
__host__ __device__ constexpr uint32_t make_idesc(int M, int N, bool a_mn, bool b_mn, bool a_bf16, bool b_bf16) {
  return (1u << 4) | ((a_bf16 ? 1u : 0u) << 7) | ((b_bf16 ? 1u : 0u) << 10) | ((a_mn ? 1u : 0u) << 15) |
         ((b_mn ? 1u : 0u) << 16) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
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
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void proxy_fence() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&r)[32]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,"
      "%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
        "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]),
        "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]),
        "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
      : "r"(taddr));
}
__device__ __forceinline__ void tmem_ld4(uint32_t taddr, uint32_t (&r)[4]) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0,%1,%2,%3}, [%4];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(taddr));
}
__device__ __forceinline__ void tmem_ld1(uint32_t taddr, uint32_t& r) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x1.b32 {%0}, [%1];" : "=r"(r) : "r"(taddr));
}
__device__ __forceinline__ uint4 lds128(uint32_t a) {
  uint4 v;
  asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(a));
  return v;
}
__device__ __forceinline__ void sts128(uint32_t a, uint4 v) {
  asm volatile("st.shared.v4.u32 [%0], {%1,%2,%3,%4};" ::"r"(a), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
__device__ __forceinline__ void sts16(uint32_t a, unsigned short v) {
  asm volatile("st.shared.u16 [%0], %1;" ::"r"(a), "h"(v) : "memory");
}
__device__ __forceinline__ void l2_prefetch(const void* p, uint32_t bytes) {
  asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}
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

// phi on one 16-byte chunk (8 elements) in place; `keep` = false zeroes it (rows past the window end)
template <bool BF16>
__device__ __forceinline__ void phi_chunk(uint32_t addr, bool keep) {
  uint4 x = lds128(addr);
  x.x = phi_h2<BF16>(x.x); x.y = phi_h2<BF16>(x.y); x.z = phi_h2<BF16>(x.z); x.w = phi_h2<BF16>(x.w);
  if (!keep) x = make_uint4(0u, 0u, 0u, 0u);
  sts128(addr, x);
}

// shared address of (row, 16-byte chunk of the 128-channel slab row) in a 16-row tile of two swizzled boxes
__device__ __forceinline__ uint32_t tile_addr(uint32_t base, int row, int chunk) {
  return base + (uint32_t)(((chunk >> 3) << 11) + row * 128 + (((chunk & 7) ^ (row & 7)) << 4));
}

template <bool BF16, typename T>
__global__ void __launch_bounds__(THREADS, 1)
sla_fwd_umma_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmK,
                    const __grid_constant__ CUtensorMap tmV, const T* __restrict__ qg, const T* __restrict__ kg_,
                    const T* __restrict__ vg, const int32_t* __restrict__ off, T* __restrict__ out,
                    float* __restrict__ ws, int N, int W, int H, int span) {
  extern __shared__ uint8_t dyn_smem[];
  __shared__ Ctrl ctrl;
  asm volatile("griddepcontrol.launch_dependents;");
  const uint32_t sbase = (smem_u32(dyn_smem) + 1023u) & ~1023u;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int Ctot = H * D;
  const int col0 = blockIdx.y * 128;                   // first channel of this slab
  const int h0 = blockIdx.y * HS;                      // first head of this slab
  const int R0 = blockIdx.x * span, R1 = min(R0 + span, N);

  // ---- set-up: barriers, TMEM, constant operands -------------------------------------------------------
  if (threadIdx.x == 0) {
    for (int i = 0; i < NIT; ++i) { mbar_init(smem_u32(&ctrl.item_full[i]), 1); mbar_init(smem_u32(&ctrl.item_empty[i]), 1 + KG_WARPS + QG_WARPS); }
    for (int i = 0; i < NKV; ++i) { mbar_init(smem_u32(&ctrl.kv_full[i]), 1); mbar_init(smem_u32(&ctrl.kphi[i]), KG_WARPS); mbar_init(smem_u32(&ctrl.kv_empty[i]), 1); }
    for (int i = 0; i < NQB; ++i) { mbar_init(smem_u32(&ctrl.q_full[i]), 1); mbar_init(smem_u32(&ctrl.qphi[i]), QG_WARPS); mbar_init(smem_u32(&ctrl.q_empty[i]), 1); }
    for (int i = 0; i < NSL; ++i) {
      mbar_init(smem_u32(&ctrl.state_full[i]), 1); mbar_init(smem_u32(&ctrl.region_free[i]), 8);
      mbar_init(smem_u32(&ctrl.o_full[i]), 1); mbar_init(smem_u32(&ctrl.o_drained[i]), QG_WARPS);
    }
    for (int i = 0; i < NB; ++i) { mbar_init(smem_u32(&ctrl.b_full[i]), 4); mbar_init(smem_u32(&ctrl.b_empty[i]), 1); }
    for (int i = 0; i < NPK; ++i) { mbar_init(smem_u32(&ctrl.pk_full[i]), 1); mbar_init(smem_u32(&ctrl.pk_empty[i]), 8); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == WARP_MMA) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&ctrl.tmem_base)), "n"(TMEM_COLS));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  // ones tile (B operand of the z MMA) and zeroed z tiles of the B buffers
  for (int i = threadIdx.x; i < ONES_BYTES / 16; i += THREADS)
    sts128(sbase + OFF_ONES + i * 16, make_uint4(0x3C003C00u, 0x3C003C00u, 0x3C003C00u, 0x3C003C00u));
  for (int i = threadIdx.x; i < NB * (4096 / 16); i += THREADS)
    sts128(sbase + OFF_B + (i / 256) * B_BUF + HS * BH_BYTES + (i % 256) * 16, make_uint4(0u, 0u, 0u, 0u));
  proxy_fence();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = ctrl.tmem_base;
  // nothing a previous kernel of the stream may have written (offsets, tensors, workspace, out) is touched before
  asm volatile("griddepcontrol.wait;" ::: "memory");

  if (warp == WARP_PROD) {
    // =========================== producer: window walk -> items -> TMA ===========================
    Cur it{0, 0}, kv{0, 0}, qb{0, 0}, pk{0, 0};
    auto emit = [&](int type, int s, int m, int aux) {
      if (lane == 0) {
        mbar_wait_wd(smem_u32(&ctrl.item_empty[it.slot]), it.phase ^ 1u);
        ctrl.items[it.slot] = make_int4(type, s, m, aux);
        mbar_arrive(smem_u32(&ctrl.item_full[it.slot]));
      }
      advance<NIT>(it);
    };
    if (R0 < R1) {
      int wa, wl;
      warp_windows_of_rows(off, W, R0, R1 - 1, wa, wl);
      // L2 prefetch cursor over the rows this CTA is about to load (whole rows of q, k, v)
      int pf_row = max(0, R0 - 64);
      const int pf_end = min(N, R1 + 128);
      auto prefetch_to = [&](int row) {
        row = min(row, pf_end);
        while (pf_row < row) {
          const int n = min(PF_CHUNK, pf_end - pf_row);
          if (lane < 3) {
            const T* base = lane == 0 ? kg_ : (lane == 1 ? vg : qg);
            l2_prefetch(base + (size_t)pf_row * Ctot, (uint32_t)(n * Ctot * 2));
          }
          pf_row += n;
        }
      };
      prefetch_to(R0 + PF_AHEAD);
      // window walk with a 32-entry register cache of the offsets
      int wbase = wa;
      int cur = __ldg(off + min(wbase + lane, W));
      int nxt = __ldg(off + min(wbase + 31 + lane, W));
      auto bounds = [&](int w, int& s, int& e) {
        int i = w - wbase;
        if (i >= 31) {
          wbase += 31;
          cur = nxt;
          nxt = __ldg(off + min(wbase + 31 + lane, W));
          i = w - wbase;
        }
        s = __shfl_sync(0xffffffffu, cur, i);
        e = __shfl_sync(0xffffffffu, cur, i + 1);
      };
      auto load_kv = [&](int y) {   // one K/V tile of 16 rows starting at row y (lane 0)
        mbar_wait_wd(smem_u32(&ctrl.kv_empty[kv.slot]), kv.phase ^ 1u);
        const uint32_t bar = smem_u32(&ctrl.kv_full[kv.slot]);
        const uint32_t dst = sbase + OFF_KV + kv.slot * KV_SLOT;
        mbar_expect_tx(bar, KV_SLOT);
        tma_load_2d(dst, &tmK, bar, col0, y);
        tma_load_2d(dst + 2048, &tmK, bar, col0 + 64, y);
        tma_load_2d(dst + 4096, &tmV, bar, col0, y);
        tma_load_2d(dst + 6144, &tmV, bar, col0 + 64, y);
        advance<NKV>(kv);
      };
      auto load_q = [&](int y, int tiles) {   // one Q block: `tiles` tiles of 16 rows starting at row y (lane 0)
        mbar_wait_wd(smem_u32(&ctrl.q_empty[qb.slot]), qb.phase ^ 1u);
        const uint32_t bar = smem_u32(&ctrl.q_full[qb.slot]);
        const uint32_t dst = sbase + OFF_Q + qb.slot * Q_BUF;
        mbar_expect_tx(bar, (uint32_t)(tiles * TILE_BYTES));
        for (int j = 0; j < tiles; ++j) {
          tma_load_2d(dst + j * 2048, &tmQ, bar, col0, y + 16 * j);
          tma_load_2d(dst + 16384 + j * 2048, &tmQ, bar, col0 + 64, y + 16 * j);
        }
        advance<NQB>(qb);
      };
      int w = wa;
      while (w < W) {
        int s, e;
        bounds(w, s, e);
        if (s >= R1) break;
        const int m = e - s;
        if (m <= kFuseMax && s + (m >> 1) >= R1) break;                          // middle beyond the span: a later CTA's
        if (m <= 0 || (m <= kFuseMax && s + (m >> 1) < R0)) { ++w; continue; }   // empty, or an earlier CTA's
        prefetch_to(min(e, R1) + PF_AHEAD);
        if (m <= 16) {
          // pack the following whole short windows (owned, together <= 16 rows) into one tile
          const int i0 = w - wbase;
          const int e_j = __shfl_down_sync(0xffffffffu, cur, 1);
          const int mid_j = cur + ((e_j - cur) >> 1);
          const bool fits = lane >= i0 && lane < 31 && (e_j - s) <= 16 && mid_j < R1;
          const unsigned okm = __ballot_sync(0xffffffffu, fits) >> i0;
          const int cnt = __ffs(~okm) - 1;
          const int rows = __shfl_sync(0xffffffffu, cur, i0 + cnt) - s;
          const unsigned startbit = (lane > i0 && lane < i0 + cnt) ? (1u << (cur - s)) : 0u;
          const unsigned starts = __reduce_or_sync(0xffffffffu, startbit) & 0xFFFEu;
          w += cnt;
          emit(IT_PACK, s, rows, (int)starts);
          if (lane == 0) {
            mbar_wait_wd(smem_u32(&ctrl.pk_empty[pk.slot]), pk.phase ^ 1u);
            const uint32_t bar = smem_u32(&ctrl.pk_full[pk.slot]);
            const uint32_t dst = sbase + OFF_PK + pk.slot * PK_SLOT;
            mbar_expect_tx(bar, PK_SLOT);
            tma_load_2d(dst, &tmK, bar, col0, s);
            tma_load_2d(dst + 2048, &tmK, bar, col0 + 64, s);
            tma_load_2d(dst + 4096, &tmV, bar, col0, s);
            tma_load_2d(dst + 6144, &tmV, bar, col0 + 64, s);
            tma_load_2d(dst + 8192, &tmQ, bar, col0, s);
            tma_load_2d(dst + 10240, &tmQ, bar, col0 + 64, s);
          }
          advance<NPK>(pk);
          continue;
        }
        if (m <= kFuseMax) {
          emit(IT_WIN, s, m, 0);
          const int T16 = (m + 15) >> 4;
          if (lane == 0) {
            const int first = min(T16, 4);             // a few K/V tiles, then Q (never queued behind a full ring)
            for (int t = 0; t < first; ++t) load_kv(s + 16 * t);
            for (int b = 0; b * 8 < T16; ++b) load_q(s + 128 * b, min(8, T16 - 8 * b));
            for (int t = first; t < T16; ++t) load_kv(s + 16 * t);
          } else {
            for (int t = 0; t < T16; ++t) advance<NKV>(kv);
            for (int b = 0; b * 8 < T16; ++b) advance<NQB>(qb);
          }
        } else if (ws != nullptr) {   // bounded entry (no workspace): a window that breaks the promise is skipped
          const int ps = max(s, R0), pe = min(e, R1);
          if (lane == 0) reinterpret_cast<volatile int*>(ws)[0] = 1;             // tell the output kernel
          emit(IT_PIECE, ps, pe - ps, s);
          const int T16 = (pe - ps + 15) >> 4;
          if (lane == 0) {
            for (int t = 0; t < T16; ++t) load_kv(ps + 16 * t);
          } else {
            for (int t = 0; t < T16; ++t) advance<NKV>(kv);
          }
        }
        ++w;
      }
    }
    emit(IT_END, 0, 0, 0);
  } else if (warp == WARP_MMA) {
    // =========================== MMA issuer ===========================
    Cur it{0, 0}, kv{0, 0}, qb{0, 0}, rg{0, 0}, bb{0, 0};
    uint32_t od_ph = 0;                                  // parity of the next o_drained completion, per region
    constexpr uint32_t ID_STATE = make_idesc(128, 128, true, true, BF16, false);   // A = V (I/O dtype), B = phi(K) fp16
    constexpr uint32_t ID_Z = make_idesc(128, 16, true, false, false, false);      // A = phi(K), B = ones
    constexpr uint32_t ID_OUT = make_idesc(128, 16, false, false, false, false);
    const uint32_t ones = sbase + OFF_ONES;
    while (true) {
      mbar_wait_wd(smem_u32(&ctrl.item_full[it.slot]), it.phase);
      const int4 d = ctrl.items[it.slot];
      __syncwarp();
      if (lane == 0) mbar_arrive(smem_u32(&ctrl.item_empty[it.slot]));
      advance<NIT>(it);
      if (d.x == IT_END) break;
      if (d.x == IT_PACK) continue;
      const int T16 = (d.z + 15) >> 4;
      const uint32_t region = tmem + (uint32_t)(rg.slot * REGION_COLS);
      mbar_wait_wd(smem_u32(&ctrl.region_free[rg.slot]), rg.phase ^ 1u);
      for (int t = 0; t < T16; ++t) {
        mbar_wait_wd(smem_u32(&ctrl.kphi[kv.slot]), kv.phase);
        tc_fence_after();
        if (lane == 0) {
          const uint32_t ks = sbase + OFF_KV + kv.slot * KV_SLOT;
          const uint64_t dk = make_desc(ks, 2048, 1024), dv = make_desc(ks + 4096, 2048, 1024);
          umma(region, dv, dk, ID_STATE, t > 0 ? 1u : 0u);
          umma(region + 128, dk, make_desc(ones, 16, 1024), ID_Z, t > 0 ? 1u : 0u);
          umma_commit(smem_u32(&ctrl.kv_empty[kv.slot]));
        }
        __syncwarp();
        advance<NKV>(kv);
      }
      if (lane == 0) umma_commit(smem_u32(&ctrl.state_full[rg.slot]));
      __syncwarp();
      if (d.x == IT_WIN) {
        const uint32_t bbuf = sbase + OFF_B + bb.slot * B_BUF;
        mbar_wait_wd(smem_u32(&ctrl.b_full[bb.slot]), bb.phase);
        for (int b = 0; b * 8 < T16; ++b) {
          mbar_wait_wd(smem_u32(&ctrl.qphi[qb.slot]), qb.phase);
          if (b > 0) {
            mbar_wait_wd(smem_u32(&ctrl.o_drained[rg.slot]), (od_ph >> rg.slot) & 1u);
            od_ph ^= 1u << rg.slot;
          }
          tc_fence_after();
          if (lane == 0) {
            const uint32_t qs = sbase + OFF_Q + qb.slot * Q_BUF;
#pragma unroll
            for (int h = 0; h < HS; ++h)
              umma(region + 16 * h, make_desc(qs + (h >> 2) * 16384 + (h & 3) * 32, 16, 1024),
                   make_desc(bbuf + h * BH_BYTES, 16, 1024), ID_OUT, 0u);
#pragma unroll
            for (int ks = 0; ks < 8; ++ks)
              umma(region + 128, make_desc(qs + (ks >> 2) * 16384 + (ks & 3) * 32, 16, 1024),
                   make_desc(bbuf + HS * BH_BYTES + (ks >> 2) * 2048 + (ks & 3) * 32, 16, 1024), ID_OUT,
                   ks > 0 ? 1u : 0u);
            umma_commit(smem_u32(&ctrl.q_empty[qb.slot]));
            umma_commit(smem_u32(&ctrl.o_full[rg.slot]));
          }
          __syncwarp();
          advance<NQB>(qb);
        }
        if (lane == 0) umma_commit(smem_u32(&ctrl.b_empty[bb.slot]));
        __syncwarp();
        advance<NB>(bb);
      }
      advance<NSL>(rg);
    }
  } else if (warp < WARP_QG0) {
    // =========================== K group: phi(K) in place, state -> B operands ===========================
    const int kgw = warp - WARP_KG0;                     // 0..7
    const int tid_g = kgw * 32 + lane;                   // 0..255: one 16-byte chunk of a K tile each
    const int quad = warp & 3;                           // TMEM lane quadrant of this warp
    Cur it{0, 0}, kv{0, 0}, rg{0, 0}, bb{0, 0}, pk{0, 0};
    int npack = 0;
    while (true) {
      mbar_wait_wd(smem_u32(&ctrl.item_full[it.slot]), it.phase);
      const int4 d = ctrl.items[it.slot];
      __syncwarp();
      if (lane == 0) mbar_arrive(smem_u32(&ctrl.item_empty[it.slot]));
      advance<NIT>(it);
      if (d.x == IT_END) break;
      if (d.x == IT_PACK) {
        if ((npack++ & 1) == 0) {                        // even packed tiles: this group; odd: the Q group
          mbar_wait_wd(smem_u32(&ctrl.pk_full[pk.slot]), pk.phase);
          const uint32_t pb = sbase + OFF_PK + pk.slot * PK_SLOT;
          const int wid = (lane < d.z) ? __popc((unsigned)d.w & ((2u << lane) - 1u)) : -1;
          if (kgw < HS)
            quad_tile_core<D, BF16, T>([&](int r, int c) { return tile_addr(pb + 8192, r, c); },
                                       [&](int r, int c) { return tile_addr(pb, r, c); },
                                       [&](int r, int c) { return tile_addr(pb + 4096, r, c); }, kgw, d.z, wid,
                                       out + (size_t)d.y * Ctot + col0 + kgw * D, Ctot);
          __syncwarp();
          if (lane == 0) mbar_arrive(smem_u32(&ctrl.pk_empty[pk.slot]));
        }
        advance<NPK>(pk);
        continue;
      }
      const int m = d.z, T16 = (m + 15) >> 4;
      for (int t = 0; t < T16; ++t) {
        mbar_wait_wd(smem_u32(&ctrl.kv_full[kv.slot]), kv.phase);
        const int row = (tid_g & 127) >> 3;
        phi_chunk<BF16>(sbase + OFF_KV + kv.slot * KV_SLOT + tid_g * 16, 16 * t + row < m);
        proxy_fence();
        __syncwarp();
        if (lane == 0) mbar_arrive(smem_u32(&ctrl.kphi[kv.slot]));
        advance<NKV>(kv);
      }
      // the state of this item is complete when the MMA warp's commit lands
      const uint32_t region = tmem + (uint32_t)(rg.slot * REGION_COLS);
      if (kgw < 4) {
        mbar_wait_wd(smem_u32(&ctrl.state_full[rg.slot]), rg.phase);
        tc_fence_after();
        uint32_t v[32], zr;
        const uint32_t lane_base = (uint32_t)(32 * quad) << 16;
        tmem_ld32(region + lane_base + 32 * quad, v);     // columns 32q..32q+31: the diagonal blocks of heads 2q, 2q+1
        tmem_ld1(region + lane_base + 128, zr);
        tmem_wait_ld();
        const int h = 2 * quad + (lane >> 4), r = lane & 15;   // this lane = channel (h, r) of the slab
        float x[16];
#pragma unroll
        for (int p = 0; p < 16; ++p) x[p] = __uint_as_float((lane & 16) ? v[16 + p] : v[p]);   // S_h[p][r]
        const float zv = __uint_as_float(zr);                                                   // z_h[r]
        if (d.x == IT_WIN) {
          const int lg = 32 - __clz(m - 1);
          const float scale = __int_as_float((127 - lg) << 23);   // 2^-ceil(log2 m): fp16 operands stay O(1)
          mbar_wait_wd(smem_u32(&ctrl.b_empty[bb.slot]), bb.phase ^ 1u);
          const uint32_t bbuf = sbase + OFF_B + bb.slot * B_BUF;
          uint4 c0, c1;
          c0.x = pack_h2(x[0] * scale, x[1] * scale);   c0.y = pack_h2(x[2] * scale, x[3] * scale);
          c0.z = pack_h2(x[4] * scale, x[5] * scale);   c0.w = pack_h2(x[6] * scale, x[7] * scale);
          c1.x = pack_h2(x[8] * scale, x[9] * scale);   c1.y = pack_h2(x[10] * scale, x[11] * scale);
          c1.z = pack_h2(x[12] * scale, x[13] * scale); c1.w = pack_h2(x[14] * scale, x[15] * scale);
          const uint32_t rowa = bbuf + h * BH_BYTES + r * 128;
          sts128(rowa + ((0 ^ (r & 7)) << 4), c0);        // B_h[n = r][k = 0..7]
          sts128(rowa + ((1 ^ (r & 7)) << 4), c1);        // B_h[n = r][k = 8..15]
          // Bden[n = h][k = 16h + r] = z_h[r]
          const __half zh = __float2half_rn(zv * scale);
          sts16(bbuf + HS * BH_BYTES + (h >> 2) * 2048 + h * 128 + (((2 * (h & 3) + (r >> 3)) ^ (h & 7)) << 4) + (r & 7) * 2,
                __half_as_ushort(zh));
          proxy_fence();
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(smem_u32(&ctrl.b_full[bb.slot]));
        } else {
          // piece of a long window: partial state -> workspace slot of the window (fp32 atomics)
          float* slot = ws + kWsHeaderFloats +
                        ((size_t)(d.w / (kFuseMax + 1)) * H + (h0 + h)) * (size_t)((D + 1) * D);
#pragma unroll
          for (int p = 0; p < 16; ++p) atomicAdd(slot + p * D + r, x[p]);
          atomicAdd(slot + D * D + r, zv);
          tc_fence_before();
        }
      }
      if (d.x == IT_WIN) {
        advance<NB>(bb);
      } else {
        __syncwarp();
        if (lane == 0) mbar_arrive(smem_u32(&ctrl.region_free[rg.slot]));   // all 8 K warps: the region is free again
      }
      advance<NSL>(rg);
    }
  } else {
    // =========================== Q group: phi(Q) in place, epilogue ===========================
    const int qgw = warp - WARP_QG0;                     // 0..7
    const int tid_g = qgw * 32 + lane;
    const int quad = warp & 3, half = qgw >> 2;          // TMEM lane quadrant; which 4 heads this warp stores
    Cur it{0, 0}, qb{0, 0}, rg{0, 0}, pk{0, 0};
    uint32_t of_ph = 0;                                  // parity of the next o_full completion, per region
    int npack = 0;
    while (true) {
      mbar_wait_wd(smem_u32(&ctrl.item_full[it.slot]), it.phase);
      const int4 d = ctrl.items[it.slot];
      __syncwarp();
      if (lane == 0) mbar_arrive(smem_u32(&ctrl.item_empty[it.slot]));
      advance<NIT>(it);
      if (d.x == IT_END) break;
      if (d.x == IT_PACK) {
        if ((npack++ & 1) == 1) {
          mbar_wait_wd(smem_u32(&ctrl.pk_full[pk.slot]), pk.phase);
          const uint32_t pb = sbase + OFF_PK + pk.slot * PK_SLOT;
          const int wid = (lane < d.z) ? __popc((unsigned)d.w & ((2u << lane) - 1u)) : -1;
          if (qgw < HS)
            quad_tile_core<D, BF16, T>([&](int r, int c) { return tile_addr(pb + 8192, r, c); },
                                       [&](int r, int c) { return tile_addr(pb, r, c); },
                                       [&](int r, int c) { return tile_addr(pb + 4096, r, c); }, qgw, d.z, wid,
                                       out + (size_t)d.y * Ctot + col0 + qgw * D, Ctot);
          __syncwarp();
          if (lane == 0) mbar_arrive(smem_u32(&ctrl.pk_empty[pk.slot]));
        }
        advance<NPK>(pk);
        continue;
      }
      if (d.x == IT_PIECE) { advance<NSL>(rg); continue; }
      const int s = d.y, m = d.z, T16 = (m + 15) >> 4;
      const int nblk = (T16 + 7) >> 3;
      for (int b = 0; b < nblk; ++b) {
        const int tiles = min(8, T16 - 8 * b);
        mbar_wait_wd(smem_u32(&ctrl.q_full[qb.slot]), qb.phase);
        const uint32_t a0 = sbase + OFF_Q + qb.slot * Q_BUF + (tid_g >> 7) * 16384 + (tid_g & 127) * 16;
        int j = 0;
        for (; j + 1 < tiles; j += 2) {
          phi_chunk<BF16>(a0 + j * 2048, true);
          phi_chunk<BF16>(a0 + (j + 1) * 2048, true);
        }
        if (j < tiles) phi_chunk<BF16>(a0 + j * 2048, true);
        proxy_fence();
        __syncwarp();
        if (lane == 0) mbar_arrive(smem_u32(&ctrl.qphi[qb.slot]));
        advance<NQB>(qb);
      }
      const uint32_t region = tmem + (uint32_t)(rg.slot * REGION_COLS);
      for (int b = 0; b < nblk; ++b) {
        const int rows = min(128, m - 128 * b);          // valid rows of this block
        mbar_wait_wd(smem_u32(&ctrl.o_full[rg.slot]), (of_ph >> rg.slot) & 1u);
        of_ph ^= 1u << rg.slot;
        tc_fence_after();
        if (32 * quad < rows) {
          const uint32_t taddr = region + ((uint32_t)(32 * quad) << 16);
          uint32_t dn[4];
          tmem_ld4(taddr + 128 + 4 * half, dn);
          const int rib = 32 * quad + lane;              // row of the block this thread owns
          T* orow = out + (size_t)(s + 128 * b + rib) * Ctot + col0 + 64 * half;
#pragma unroll
          for (int hp = 0; hp < 2; ++hp) {               // two heads per 32-column load
            uint32_t v[32];
            tmem_ld32(taddr + 64 * half + 32 * hp, v);
            tmem_wait_ld();
            const float i0 = fast_rcp(__uint_as_float(dn[2 * hp])), i1 = fast_rcp(__uint_as_float(dn[2 * hp + 1]));
            if (rib < rows) {
              uint4 o0, o1, o2, o3;
              o0.x = pack_out<BF16>(__uint_as_float(v[0]) * i0, __uint_as_float(v[1]) * i0);
              o0.y = pack_out<BF16>(__uint_as_float(v[2]) * i0, __uint_as_float(v[3]) * i0);
              o0.z = pack_out<BF16>(__uint_as_float(v[4]) * i0, __uint_as_float(v[5]) * i0);
              o0.w = pack_out<BF16>(__uint_as_float(v[6]) * i0, __uint_as_float(v[7]) * i0);
              o1.x = pack_out<BF16>(__uint_as_float(v[8]) * i0, __uint_as_float(v[9]) * i0);
              o1.y = pack_out<BF16>(__uint_as_float(v[10]) * i0, __uint_as_float(v[11]) * i0);
              o1.z = pack_out<BF16>(__uint_as_float(v[12]) * i0, __uint_as_float(v[13]) * i0);
              o1.w = pack_out<BF16>(__uint_as_float(v[14]) * i0, __uint_as_float(v[15]) * i0);
              o2.x = pack_out<BF16>(__uint_as_float(v[16]) * i1, __uint_as_float(v[17]) * i1);
              o2.y = pack_out<BF16>(__uint_as_float(v[18]) * i1, __uint_as_float(v[19]) * i1);
              o2.z = pack_out<BF16>(__uint_as_float(v[20]) * i1, __uint_as_float(v[21]) * i1);
              o2.w = pack_out<BF16>(__uint_as_float(v[22]) * i1, __uint_as_float(v[23]) * i1);
              o3.x = pack_out<BF16>(__uint_as_float(v[24]) * i1, __uint_as_float(v[25]) * i1);
              o3.y = pack_out<BF16>(__uint_as_float(v[26]) * i1, __uint_as_float(v[27]) * i1);
              o3.z = pack_out<BF16>(__uint_as_float(v[28]) * i1, __uint_as_float(v[29]) * i1);
              o3.w = pack_out<BF16>(__uint_as_float(v[30]) * i1, __uint_as_float(v[31]) * i1);
              uint4* op = reinterpret_cast<uint4*>(orow + 32 * hp);
              op[0] = o0; op[1] = o1; op[2] = o2; op[3] = o3;
            }
          }
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0)
          mbar_arrive(smem_u32(b + 1 < nblk ? &ctrl.o_drained[rg.slot] : &ctrl.region_free[rg.slot]));
      }
      advance<NSL>(rg);
    }
  }

  // ---- teardown ---------------------------------------------------------------------------------------
  tc_fence_before();
  __syncthreads();
  if (warp == WARP_MMA) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(TMEM_COLS));
  }
}

// 2-D map over a row-major [N, C] 16-bit tensor; box = 64 columns (128 B) x 16 rows, 128-byte swizzle
template <bool BF16, typename T>
cudaError_t umma_launch(const Problem& p, cudaStream_t st) {
  CUtensorMap tq, tk, tv;
  const int Ctot = p.H * D;
  if (!make_map(&tq, p.q, p.N, Ctot, 16) || !make_map(&tk, p.k, p.N, Ctot, 16) || !make_map(&tv, p.v, p.N, Ctot, 16))
    return cudaErrorInvalidValue;
  auto kern = sla_fwd_umma_kernel<BF16, T>;
  static std::atomic<bool> attr_set[kMaxDevices];         // the smem opt-in is per device
  const int dev = current_device();
  if (!attr_set[dev].load(std::memory_order_acquire)) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_DYN);
    if (e != cudaSuccess) return e;
    attr_set[dev].store(true, std::memory_order_release);
  }
  const int slabs = Ctot / 128;
  int nx = sm_count() / slabs;                             // one persistent CTA per SM
  if (nx < 1) nx = 1;
  int span = (p.N + nx - 1) / nx;
  if (span < 64) span = 64;
  nx = (p.N + span - 1) / span;
  cudaLaunchAttribute pdl[1];
  pdl[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  pdl[0].val.programmaticStreamSerializationAllowed = 1;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(nx, slabs);
  cfg.blockDim = dim3(THREADS);
  cfg.dynamicSmemBytes = SMEM_DYN;
  cfg.stream = st;
  cfg.attrs = pdl;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kern, tq, tk, tv, (const T*)p.q, (const T*)p.k, (const T*)p.v, p.off, (T*)p.out,
                            p.ws_state, p.N, p.W, p.H, span);
}

}  // namespace

bool forward_umma_supported(const Problem& p, int dt) {
  if (dt != SLA_F16) return false;
  if (p.d != D || (p.H * p.d) % 128 != 0) return false;
  return encode_fn() != nullptr;
}

cudaError_t launch_forward_umma_main(const Problem& p, int dt, cudaStream_t st) {
  (void)dt;
  return umma_launch<false, __half>(p, st);
}

}  // namespace sla
