// sla_fwd_umma.cu -- SLA forward on the 5th-generation tensor cores (tcgen05.mma, accumulators in TMEM), all heads
// of a 128-channel slab at once.  fp16 I/O, d_h = 16, H*d_h a multiple of 128.
//
// What is computed (Eq. 2-3): per window w and head h
//     S = sum_j phi(k_j)^T v_j,   z = sum_j phi(k_j),   o_i = phi(q_i) S / (phi(q_i) . z).
//
// Design (parity-tested entry sla_forward_tcgen05, not the default path):
//   * One persistent CTA per SM; the flat window-sorted matrix is cut into one row span per CTA
//     (load balance by rows, Fig. 3a).  A CTA owns every window of <= kFuseMax rows whose middle
//     row lies in its span, and the pieces of longer windows that intersect it (partial state -> fp32 atomics
//     into the workspace; their outputs come from the OUTPASS launch of sla_fwd_tc.cu).
//   * The walk warp turns the window offsets into ITEMS (a descriptor ring in shared memory):
//       PACK   consecutive whole windows of <= 16 rows, together <= 16 rows: one packed tile, masked quadratic
//              form on mma.sync with split operands (quad_tile_core) -- the fp16-operand linear form does not
//              meet the tolerance on windows this short;
//       WIN    one window of 17..kFuseMax rows;
//       PIECE  the part of a longer window inside this span (state only).
//     Rows travel in CHUNKS of one item: the walk warp loads K,V chunks of <= 4 tiles of 16 rows, a second loader
//     warp Q chunks of <= 8 tiles (one MMA block of up to 128 rows), with 2-D TMA boxes of 64 channels x
//     16/32/64/128 rows (128-byte swizzle) into tile rings; a chunk never wraps around its ring.
//   * 8 phi warps (one 16-byte chunk of every tile of the chunk per thread) apply phi to K and Q tiles IN PLACE
//     (K rows past the window end are zeroed: the contraction of the state MMA runs over rows).
//   * The state issuer warp then runs, per 16 rows and straight from the TMA tiles,
//         D[r][p]  += sum_j V[j][r] phi(K)[j][p]      tcgen05.mma M=128 N=128 K=16, both operands MN-major,
//         Z[p][.]  += sum_j phi(K)[j][p] * 1          tcgen05.mma M=128 N=16  K=16 against a tile of ones.
//     The 16x16 diagonal blocks of D are the per-head states S_h^T; the off-diagonal blocks (7/8 of the tensor
//     work, ~64 cycles per 16 rows) are ignored.
//   * When a window's state is complete the convert warps read its diagonal blocks and z from TMEM, scale them by
//     2^-ceil(log2 m) (Eq. 3 is a ratio) and write them as fp16 B operands: per head a [32 x 16] K-major tile,
//     rows 0..15 = S_h[.][r], row 16 = z_h.
//   * The output issuer runs per head  O[i][32h..32h+31] = phi(Q)[i][16h..16h+15] . B_h^T  (M=128 N=32 K=16):
//     columns 32h..32h+15 are the numerators, column 32h+16 the denominator, in the TMEM columns the state
//     occupied.  Epilogue warps read their rows back (one thread per row), divide, stage the fp16 rows in the
//     (now dead) Q tiles and store them with fully coalesced 128-bit stores.
//   * Barrier discipline: ring barriers are indexed by the first tile of a chunk; a role that waits on a barrier
//     family waits on it at every use (a role that only toggled a parity could run a phase ahead and pass a
//     try_wait.parity on the wrong phase), and barriers that complete only for some item types (kphi, qphi) have their
//     own parity bits.
//   * Precision: operands fp16, accumulation fp32.
#include <cuda.h>

#include <atomic>
#include <cstdio>

#include "sla_internal.cuh"

namespace sla {
namespace {

#include "sla_tc_base.cuh"

constexpr int D = 16;                       // head dim of this kernel
constexpr int HS = 128 / D;                 // heads per 128-channel slab
constexpr int NKV = 14;                     // K/V tile ring (tiles of 16 rows: K 4 KB + V 4 KB, as four 64-channel box regions)
constexpr int NQT = 18;                     // Q tile ring (4 KB per tile, as two box regions)
constexpr int NSL = 2;                      // TMEM regions of 256 columns (state, then output, of one item)
constexpr int NB = 3;                       // B operand buffers (2 tiles of 4 heads x 32 rows = 8 KB)
constexpr int NIT = 16;                     // item descriptor ring
constexpr int KVC = 4;                      // tiles per K/V chunk (Q chunks are MMA blocks of up to 8 tiles)
#ifndef SLA_NEPI
#define SLA_NEPI 4
#endif
constexpr int NPHI = 8, NCONV = 4, NEPI = SLA_NEPI;      // NEPI = 4: each epilogue warp stores all 8 heads of its 32 rows
constexpr int EPI_HALVES = 8 / NEPI;
constexpr int WARP_WALK = 0, WARP_QLOAD = 1, WARP_SMMA = 2, WARP_OMMA = 3, WARP_PHI0 = 4,
              WARP_CONV0 = WARP_PHI0 + NPHI, WARP_EPI0 = WARP_CONV0 + NCONV, NWARPS = WARP_EPI0 + NEPI;
constexpr int THREADS = NWARPS * 32;
constexpr int NREADERS = NWARPS - 1;        // every warp but the walk warp reads the item ring
constexpr int KV_REG = NKV * 2048, Q_REG = NQT * 2048;          // one 64-channel box region of a ring
constexpr int B_BUF = 2 * 4096, ONES_BYTES = 2048;
constexpr int OFF_K = 0, OFF_V = 2 * KV_REG, OFF_Q = 4 * KV_REG, OFF_B = OFF_Q + 2 * Q_REG, OFF_ONES = OFF_B + NB * B_BUF;
constexpr int SMEM_DYN = OFF_ONES + ONES_BYTES + 1024;          // + alignment slack (swizzle needs 1 KB)
constexpr int REGION_COLS = 256, TMEM_COLS = 512;
constexpr int PF_FIRST = 1024, PF_CHUNK = 32;                   // L2 prefetch: rows requested up front / per request
static_assert(NB * B_BUF >= 7 * 2048, "an M=128 Q block starting at the last ring tile reads 7 tiles past the ring");
static_assert(NKV <= 32 && NQT <= 32, "one parity bit per ring tile");


enum ItemType { IT_END = 0, IT_PACK = 1, IT_WIN = 2, IT_PIECE = 3 };

// Barriers.  Ring barriers are indexed by the FIRST tile of a chunk and complete one phase per use of that index.
struct Ctrl {
  unsigned long long item_full[NIT], item_empty[NIT];
  unsigned long long kv_full[NKV], kphi[NKV], kv_empty[NKV];
  unsigned long long q_full[NQT], qphi[NQT], q_empty[NQT];
  unsigned long long state_full[NSL], region_free[NSL], o_full[NSL], o_drained[NSL];
  unsigned long long b_full[NB], b_empty[NB];
  int4 items[NIT];
  uint32_t tmem_base;
  int search_lo;
  int kv_owner[NKV], q_owner[NQT];         // loader-private: the chunk (first tile) that last used each tile, or -1
};

struct Cur {                                 // ring cursor: slot and the parity of the current use of that slot
  int slot;
  uint32_t phase;
};
template <int N>
__device__ __forceinline__ void advance(Cur& c) {
  if (++c.slot == N) { c.slot = 0; c.phase ^= 1u; }
}
// Tile ring with contiguous chunk allocation: a chunk of n tiles never wraps (its tiles are one MMA operand); tiles
// skipped at the end of the ring are not used in that round.  Every role keeps one parity bit per chunk barrier index.
template <int N>
struct TileRing {
  int pos;
  uint32_t bits;
  __device__ __forceinline__ int alloc(int n) {
    if (pos + n > N) pos = 0;
    const int first = pos;
    pos += n;
    return first;
  }
  __device__ __forceinline__ uint32_t parity(int t) const { return (bits >> t) & 1u; }
  __device__ __forceinline__ void used(int t) { bits ^= 1u << t; }
};

struct Maps { CUtensorMap m[3][4]; };        // [q, k, v][box rows 16, 32, 64, 128]

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

__device__ __forceinline__ void mbar_arrive_relaxed(uint32_t bar) {
  asm volatile("mbarrier.arrive.relaxed.cta.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_n(uint32_t bar, uint32_t n) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(n) : "memory");
}

__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&r)[16]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
        "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
      : "r"(taddr));
}

// phi in place on the 8 sixteen-byte chunks a lane owns of one tile (chunk c at addr[c]); keep_mask bit c = 0 zeroes
// chunk c (rows past the window end).  All loads are issued before the first use.
template <bool BF16>
__device__ __forceinline__ void phi_tile_lane(const uint32_t (&addr)[8], uint32_t keep_mask) {
  uint4 x[8];
#pragma unroll
  for (int c = 0; c < 8; ++c) x[c] = lds128(addr[c]);
#pragma unroll
  for (int c = 0; c < 8; ++c) {
    x[c].x = phi_h2<BF16>(x[c].x); x[c].y = phi_h2<BF16>(x[c].y);
    x[c].z = phi_h2<BF16>(x[c].z); x[c].w = phi_h2<BF16>(x[c].w);
    if (!((keep_mask >> c) & 1u)) x[c] = make_uint4(0u, 0u, 0u, 0u);
    sts128(addr[c], x[c]);
  }
}
// the 8 chunk addresses of a lane in ring tile t (box regions box0, box0 + reg): chunk c -> region c/4, chunk
// (lane + 32 (c%4)) of the 2 KB box tile, i.e. tile row (lane/8) + 4 (c%4)
__device__ __forceinline__ void lane_chunks(uint32_t box0, int reg, int t, uint32_t (&addr)[8]) {
  const uint32_t a = box0 + (uint32_t)(t * 2048 + (threadIdx.x & 31) * 16);
#pragma unroll
  for (int c = 0; c < 8; ++c) addr[c] = a + (uint32_t)((c >> 2) * reg + (c & 3) * 512);
}
// shared address of (row, 16-byte chunk of the 128-channel slab row) in a 16-row tile whose two swizzled
// 64-channel boxes start at box0 and box1
__device__ __forceinline__ uint32_t tile_addr(uint32_t box0, uint32_t box1, int row, int chunk) {
  return ((chunk >> 3) ? box1 : box0) + (uint32_t)(row * 128 + (((chunk & 7) ^ (row & 7)) << 4));
}

template <bool BF16, typename T>
__global__ void __launch_bounds__(THREADS, 1)
sla_fwd_umma_kernel(const __grid_constant__ Maps maps, const T* __restrict__ qg, const T* __restrict__ kg_,
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
  {
    const int t = threadIdx.x;
    if (t < NIT) { mbar_init(smem_u32(&ctrl.item_full[t]), 1); mbar_init(smem_u32(&ctrl.item_empty[t]), NREADERS); }
    if (t < NKV) {
      mbar_init(smem_u32(&ctrl.kv_full[t]), 1); mbar_init(smem_u32(&ctrl.kphi[t]), 8); mbar_init(smem_u32(&ctrl.kv_empty[t]), 1);
      ctrl.kv_owner[t] = -1;
    }
    if (t < NQT) {
      mbar_init(smem_u32(&ctrl.q_full[t]), 1); mbar_init(smem_u32(&ctrl.qphi[t]), 8); mbar_init(smem_u32(&ctrl.q_empty[t]), NEPI);
      ctrl.q_owner[t] = -1;
    }
    if (t < NSL) {
      mbar_init(smem_u32(&ctrl.state_full[t]), 1); mbar_init(smem_u32(&ctrl.region_free[t]), NEPI);
      mbar_init(smem_u32(&ctrl.o_full[t]), 1); mbar_init(smem_u32(&ctrl.o_drained[t]), NEPI);
    }
    if (t < NB) { mbar_init(smem_u32(&ctrl.b_full[t]), NCONV); mbar_init(smem_u32(&ctrl.b_empty[t]), 1); }
    if (t == 0) ctrl.search_lo = 0;
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == WARP_SMMA) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&ctrl.tmem_base)), "n"(TMEM_COLS));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  if (warp == WARP_WALK && lane < 12)
    asm volatile("prefetch.tensormap [%0];" ::"l"(&maps.m[lane >> 2][lane & 3]) : "memory");
  // ones tile (B operand of the z MMA)
  for (int i = threadIdx.x; i < ONES_BYTES / 16; i += THREADS)
    sts128(sbase + OFF_ONES + i * 16, make_uint4(0x3C003C00u, 0x3C003C00u, 0x3C003C00u, 0x3C003C00u));
  proxy_fence();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = ctrl.tmem_base;
  // nothing a previous kernel of the stream may have written (offsets, tensors, workspace, out) is touched before
  asm volatile("griddepcontrol.wait;" ::: "memory");
  // the rows of this span go to L2 now, in the order they will be needed (whole rows of k, v, q)
  if (warp == WARP_WALK && lane < 3 && R0 < R1) {
    const T* base = lane == 0 ? kg_ : (lane == 1 ? vg : qg);
    const int lo = max(0, R0 - 64), hi = min(N, min(R1 + 128, lo + PF_FIRST));
    for (int r = lo; r < hi; r += PF_CHUNK)
      l2_prefetch(base + (size_t)r * Ctot, (uint32_t)(min(PF_CHUNK, hi - r) * Ctot * 2));
  }
  // first round of the window search by the whole CTA: the largest probe idx with off[idx] <= R0
  const int sstep = (W + THREADS - 1) / THREADS;
  if (R0 < R1) {
    const long long idx = (long long)(threadIdx.x + 1) * sstep;
    if (idx < W && __ldg(off + idx) <= R0) atomicMax(&ctrl.search_lo, (int)idx);
  }
  __syncthreads();
  // every consumer role reads the item ring in order
  auto next_item = [&](Cur& it) -> int4 {
    mbar_wait_wd(smem_u32(&ctrl.item_full[it.slot]), it.phase);
    const int4 d = ctrl.items[it.slot];
    __syncwarp();
    if (lane == 0) mbar_arrive(smem_u32(&ctrl.item_empty[it.slot]));
    advance<NIT>(it);
    return d;
  };
  // Loader side of a tile ring (lane 0): make tiles [first, first+n) reusable.  A tile is guarded by the empty barrier
  // of the chunk that last used it (indexed by that chunk's first tile); its parity is that of the index's last use.
  auto claim_tiles = [&](int* owner, unsigned long long* empty, int ntiles, uint32_t bits, int first, int n) {
    for (int t = first; t < first + n; ++t) {
      const int o = owner[t];
      if (o >= 0) {
        mbar_wait_wd(smem_u32(&empty[o]), ((bits >> o) & 1u) ^ 1u);
        for (int u = 0; u < ntiles; ++u)
          if (owner[u] == o) owner[u] = -1;
      }
    }
    for (int t = first; t < first + n; ++t) owner[t] = first;
  };
  // a chunk of n tiles as boxes of 8 / 4 / 2 / 1 tiles: op(map index, first row, first tile)
  auto for_pieces = [&](int n, int y, int tile, auto&& op) {
#pragma unroll
    for (int k = 3; k >= 0; --k)
      if (n & (1 << k)) { op(k, y, tile); y += 16 << k; tile += 1 << k; }
  };

  if (warp == WARP_WALK) {
    // =========================== walk: window offsets -> items; K,V chunk loads ===========================
    Cur it{0, 0};
    TileRing<NKV> kr{0, 0u};
    auto emit = [&](int type, int s, int m, int aux) {
      if (lane == 0) {
        mbar_wait_wd(smem_u32(&ctrl.item_empty[it.slot]), it.phase ^ 1u);
        ctrl.items[it.slot] = make_int4(type, s, m, aux);
        mbar_arrive(smem_u32(&ctrl.item_full[it.slot]));
      }
      advance<NIT>(it);
    };
    if (R0 < R1) {
      // second round of the search: off[lo] <= R0 < off[min(W, lo + sstep)]
      int lo = ctrl.search_lo, hi = min(W, lo + sstep);
      while (hi - lo > 1) {
        const int step = max(1, (hi - lo + 31) / 32);
        const int idx = lo + (lane + 1) * step;
        const bool ok = idx < hi && __ldg(off + min(idx, W)) <= R0;
        const int cnt = __popc(__ballot_sync(0xffffffffu, ok));
        lo += cnt * step;
        hi = min(hi, lo + step);
      }
      const int wa = lo;
      int pf_row = min(N, min(R1 + 128, max(0, R0 - 64) + PF_FIRST));
      const int pf_end = min(N, R1 + 128);
      auto prefetch_to = [&](int row) {       // rows beyond the first PF_FIRST: requested as the walk advances
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
      auto load_kv = [&](int y, int T16) {   // the K,V tiles of rows [y, y + 16 T16) in chunks of <= KVC tiles
        for (int c = 0; c * KVC < T16; ++c) {
          const int n = min(KVC, T16 - KVC * c);
          const int first = kr.alloc(n);
          if (lane == 0) {
            claim_tiles(ctrl.kv_owner, ctrl.kv_empty, NKV, kr.bits, first, n);
            const uint32_t bar = smem_u32(&ctrl.kv_full[first]);
            mbar_expect_tx(bar, (uint32_t)(n * 8192));
            for_pieces(n, y + 16 * KVC * c, first, [&](int mi, int yy, int tile) {
              const uint32_t dk = sbase + OFF_K + tile * 2048, dv = sbase + OFF_V + tile * 2048;
              tma_load_2d(dk, &maps.m[1][mi], bar, col0, yy);
              tma_load_2d(dk + KV_REG, &maps.m[1][mi], bar, col0 + 64, yy);
              tma_load_2d(dv, &maps.m[2][mi], bar, col0, yy);
              tma_load_2d(dv + KV_REG, &maps.m[2][mi], bar, col0 + 64, yy);
            });
          }
          kr.used(first);
        }
      };
      int w = wa;
      while (w < W) {
        int s, e;
        bounds(w, s, e);
        if (s >= R1) break;
        const int m = e - s;
        if (m <= kFuseMax && s + (m >> 1) >= R1) break;                          // middle beyond the span: a later CTA's
        if (m <= 0 || (m <= kFuseMax && s + (m >> 1) < R0)) { ++w; continue; }   // empty, or an earlier CTA's
        prefetch_to(min(e, R1) + PF_FIRST / 2);
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
          load_kv(s, 1);
          continue;
        }
        if (m <= kFuseMax) {
          emit(IT_WIN, s, m, 0);
          load_kv(s, (m + 15) >> 4);
        } else if (ws != nullptr) {   // bounded entry (no workspace): a window that breaks the promise is skipped
          const int ps = max(s, R0), pe = min(e, R1);
          if (lane == 0) reinterpret_cast<volatile int*>(ws)[0] = 1;             // tell the output kernel
          emit(IT_PIECE, ps, pe - ps, s);
          load_kv(ps, (pe - ps + 15) >> 4);
        }
        ++w;
      }
    }
    emit(IT_END, 0, 0, 0);
  } else if (warp == WARP_QLOAD) {
    // =========================== Q chunk loads ===========================
    Cur it{0, 0};
    TileRing<NQT> qr{0, 0u};
    while (true) {
      const int4 d = next_item(it);
      if (d.x == IT_END) break;
      if (d.x == IT_PIECE) continue;
      const int T16 = d.x == IT_PACK ? 1 : (d.z + 15) >> 4;
      for (int c = 0; c * 8 < T16; ++c) {
        const int n = min(8, T16 - 8 * c);
        const int first = qr.alloc(n);
        if (lane == 0) {
          claim_tiles(ctrl.q_owner, ctrl.q_empty, NQT, qr.bits, first, n);
          const uint32_t bar = smem_u32(&ctrl.q_full[first]);
          mbar_expect_tx(bar, (uint32_t)(n * 4096));
          for_pieces(n, d.y + 128 * c, first, [&](int mi, int yy, int tile) {
            const uint32_t dq = sbase + OFF_Q + tile * 2048;
            tma_load_2d(dq, &maps.m[0][mi], bar, col0, yy);
            tma_load_2d(dq + Q_REG, &maps.m[0][mi], bar, col0 + 64, yy);
          });
        }
        qr.used(first);
      }
    }
  } else if (warp == WARP_SMMA) {
    // =========================== state MMA issuers: D += V^T phi(K)  |  Z += phi(K)^T 1 ===========================
    Cur it{0, 0}, rg{0, 0};
    TileRing<NKV> kr{0, 0u};
    constexpr uint32_t ID_STATE = make_idesc(128, 128, true, true, BF16, false);   // A = V (I/O dtype), B = phi(K) fp16
    constexpr uint32_t ID_Z = make_idesc(128, 16, true, false, false, false);      // A = phi(K), B = ones
    const uint64_t dones = make_desc(sbase + OFF_ONES, 16, 1024);
    uint32_t kphi_bits = 0;   // kphi completes a phase only for chunks that pass through the MMA: its own parity bits
    while (true) {
      const int4 d = next_item(it);
      if (d.x == IT_END) break;
      if (d.x == IT_PACK) { kr.alloc(1); continue; }     // a packed tile passes through no MMA: ring position only
      const int T16 = (d.z + 15) >> 4;
      const uint32_t region = tmem + (uint32_t)(rg.slot * REGION_COLS);
      mbar_wait_wd(smem_u32(&ctrl.region_free[rg.slot]), rg.phase ^ 1u);
      for (int c = 0; c * KVC < T16; ++c) {
        const int n = min(KVC, T16 - KVC * c);
        const int first = kr.alloc(n);
        mbar_wait_wd(smem_u32(&ctrl.kphi[first]), (kphi_bits >> first) & 1u);
        kphi_bits ^= 1u << first;
        tc_fence_after();
        if (lane == 0) {
          for (int j = 0; j < n; ++j) {
            const uint32_t kt = sbase + OFF_K + (first + j) * 2048;
            const uint64_t dk = make_desc(kt, KV_REG, 1024);
            const uint32_t acc = (c | j) ? 1u : 0u;
            umma(region, make_desc(kt + (OFF_V - OFF_K), KV_REG, 1024), dk, ID_STATE, acc);
            umma(region + 128, dk, dones, ID_Z, acc);
          }
          umma_commit(smem_u32(&ctrl.kv_empty[first]));
        }
        __syncwarp();
      }
      if (lane == 0) umma_commit(smem_u32(&ctrl.state_full[rg.slot]));
      __syncwarp();
      advance<NSL>(rg);
    }
  } else if (warp == WARP_OMMA) {
    // =========================== output MMA issuer ===========================
    Cur it{0, 0}, rg{0, 0}, bb{0, 0};
    TileRing<NQT> qr{0, 0u};
    uint32_t od_ph = 0;                                  // parity of the next o_drained completion, per region
    uint32_t qphi_bits = 0;                              // qphi completes a phase only for chunks of WIN items
    constexpr uint32_t ID_OUT = make_idesc(128, 32, false, false, false, false);
    while (true) {
      const int4 d = next_item(it);
      if (d.x == IT_END) break;
      if (d.x == IT_PACK) { qr.alloc(1); continue; }
      if (d.x == IT_PIECE) { advance<NSL>(rg); continue; }
      const int T16 = (d.z + 15) >> 4;
      const uint32_t region = tmem + (uint32_t)(rg.slot * REGION_COLS);
      const uint32_t bbuf = sbase + OFF_B + bb.slot * B_BUF;
      mbar_wait_wd(smem_u32(&ctrl.b_full[bb.slot]), bb.phase);
      for (int b = 0; b * 8 < T16; ++b) {
        const int n = min(8, T16 - 8 * b);
        const int first = qr.alloc(n);
        mbar_wait_wd(smem_u32(&ctrl.qphi[first]), (qphi_bits >> first) & 1u);
        qphi_bits ^= 1u << first;
        if (b > 0) {
          mbar_wait_wd(smem_u32(&ctrl.o_drained[rg.slot]), (od_ph >> rg.slot) & 1u);
          od_ph ^= 1u << rg.slot;
        }
        tc_fence_after();
        if (lane == 0) {
          const uint32_t qs0 = sbase + OFF_Q + first * 2048;
#pragma unroll
          for (int h = 0; h < HS; ++h)
            umma(region + 32 * h, make_desc(qs0 + (h >> 2) * Q_REG + (h & 3) * 32, 16, 1024),
                 make_desc(bbuf + (h >> 2) * 4096 + (h & 3) * 32, 16, 1024), ID_OUT, 0u);
          umma_commit(smem_u32(&ctrl.o_full[rg.slot]));
        }
        __syncwarp();
      }
      if (lane == 0) umma_commit(smem_u32(&ctrl.b_empty[bb.slot]));
      __syncwarp();
      advance<NB>(bb);
      advance<NSL>(rg);
    }
  } else if (warp < WARP_CONV0) {
    // =========================== phi warps: all 256 threads on every chunk, one 16-byte chunk of each tile per thread ===========
    const int pw = warp - WARP_PHI0;
    const int tid_g = pw * 32 + lane;                    // 16-byte chunk of a 4 KB tile: box region tid_g/128, row (tid_g%128)/8
    const uint32_t coff = (uint32_t)((tid_g & 127) * 16);
    const int crow = (tid_g & 127) >> 3;
    Cur it{0, 0};
    TileRing<NKV> kr{0, 0u};
    TileRing<NQT> qr{0, 0u};
    // phi in place on this thread's chunk of tiles first .. first+n-1 (n <= 4 at a time: the loads go out together)
    auto phi_chunk = [&](uint32_t base, int first, int n, int row0, int m) {
      for (int j0 = 0; j0 < n; j0 += 4) {
        uint4 x[4];
#pragma unroll
        for (int j = 0; j < 4; ++j)
          if (j0 + j < n) x[j] = lds128(base + (first + j0 + j) * 2048 + coff);
#pragma unroll
        for (int j = 0; j < 4; ++j)
          if (j0 + j < n) {
            x[j].x = phi_h2<BF16>(x[j].x); x[j].y = phi_h2<BF16>(x[j].y);
            x[j].z = phi_h2<BF16>(x[j].z); x[j].w = phi_h2<BF16>(x[j].w);
            if (row0 + 16 * (j0 + j) + crow >= m) x[j] = make_uint4(0u, 0u, 0u, 0u);   // rows past the window end
            sts128(base + (first + j0 + j) * 2048 + coff, x[j]);
          }
      }
    };
    while (true) {
      const int4 d = next_item(it);
      if (d.x == IT_END) break;
      if (d.x == IT_PACK) {
        const int kt = kr.alloc(1), qt = qr.alloc(1);
        mbar_wait_wd(smem_u32(&ctrl.kv_full[kt]), kr.parity(kt));
        mbar_wait_wd(smem_u32(&ctrl.q_full[qt]), qr.parity(qt));
        const uint32_t kb = sbase + OFF_K + kt * 2048, vb = sbase + OFF_V + kt * 2048, qb = sbase + OFF_Q + qt * 2048;
        const int wid = (lane < d.z) ? __popc((unsigned)d.w & ((2u << lane) - 1u)) : -1;
        if (pw < HS)                                     // warp pw = head pw of the slab
          quad_tile_core<D, BF16, T>([&](int r, int c) { return tile_addr(qb, qb + Q_REG, r, c); },
                                     [&](int r, int c) { return tile_addr(kb, kb + KV_REG, r, c); },
                                     [&](int r, int c) { return tile_addr(vb, vb + KV_REG, r, c); }, pw, d.z, wid,
                                     out + (size_t)d.y * Ctot + col0 + pw * D, Ctot);
        asm volatile("bar.sync 1, %0;" ::"n"(NPHI * 32) : "memory");   // every head is done with the tiles
        if (tid_g == 0) {
          mbar_arrive_n(smem_u32(&ctrl.kv_empty[kt]), 1);
          mbar_arrive_n(smem_u32(&ctrl.q_empty[qt]), NEPI);
        }
        kr.used(kt);
        qr.used(qt);
        continue;
      }
      const int m = d.z, T16 = (m + 15) >> 4;
      for (int c = 0; c * KVC < T16; ++c) {
        const int n = min(KVC, T16 - KVC * c);
        const int first = kr.alloc(n);
        mbar_wait_wd(smem_u32(&ctrl.kv_full[first]), kr.parity(first));
        phi_chunk(sbase + OFF_K + (tid_g >> 7) * KV_REG, first, n, 16 * KVC * c, m);
        proxy_fence();
        __syncwarp();
        if (lane == 0) mbar_arrive(smem_u32(&ctrl.kphi[first]));
        kr.used(first);
      }
      if (d.x == IT_WIN) {
        for (int b = 0; b * 8 < T16; ++b) {
          const int n = min(8, T16 - 8 * b);
          const int first = qr.alloc(n);
          mbar_wait_wd(smem_u32(&ctrl.q_full[first]), qr.parity(first));
          phi_chunk(sbase + OFF_Q + (tid_g >> 7) * Q_REG, first, n, 0, 1 << 30);
          proxy_fence();
          __syncwarp();
          if (lane == 0) mbar_arrive(smem_u32(&ctrl.qphi[first]));
          qr.used(first);
        }
      }
    }
  } else if (warp < WARP_EPI0) {
    // =========================== state -> B operands (or workspace atomics for pieces) ===========================
    const int quad = warp & 3;                           // TMEM lane quadrant of this warp
    Cur it{0, 0}, rg{0, 0}, bb{0, 0};
    while (true) {
      const int4 d = next_item(it);
      if (d.x == IT_END) break;
      if (d.x == IT_PACK) continue;
      const int m = d.z;
      const uint32_t region = tmem + (uint32_t)(rg.slot * REGION_COLS);
      mbar_wait_wd(smem_u32(&ctrl.state_full[rg.slot]), rg.phase);
      tc_fence_after();
      uint32_t v[32], zr;
      const uint32_t lane_base = (uint32_t)(32 * quad) << 16;
      tmem_ld32(region + lane_base + 32 * quad, v);       // columns 32q..32q+31: the diagonal blocks of heads 2q, 2q+1
      tmem_ld1(region + lane_base + 128, zr);
      tmem_wait_ld();
      const int h = 2 * quad + (lane >> 4), r = lane & 15;     // this lane = channel (h, r) of the slab
      float x[16];
#pragma unroll
      for (int p = 0; p < 16; ++p) x[p] = __uint_as_float((lane & 16) ? v[16 + p] : v[p]);   // S_h[p][r]
      const float zv = __uint_as_float(zr);                                                   // z_h[r]
      if (d.x == IT_WIN) {
        // power of two that brings the head's largest z into [1, 2) (as sla_fwd_tc.cu: state_scale); the 16 lanes of a
        // head hold z_h[0..15]
        float zm = zv;
#pragma unroll
        for (int o = 1; o < 16; o <<= 1) zm = fmaxf(zm, __shfl_xor_sync(0xffffffffu, zm, o));
        const float scale = __int_as_float((254 - ((__float_as_int(zm) >> 23) & 0xff)) << 23);
        mbar_wait_wd(smem_u32(&ctrl.b_empty[bb.slot]), bb.phase ^ 1u);
        uint4 c0, c1;
        c0.x = pack_h2(x[0] * scale, x[1] * scale);   c0.y = pack_h2(x[2] * scale, x[3] * scale);
        c0.z = pack_h2(x[4] * scale, x[5] * scale);   c0.w = pack_h2(x[6] * scale, x[7] * scale);
        c1.x = pack_h2(x[8] * scale, x[9] * scale);   c1.y = pack_h2(x[10] * scale, x[11] * scale);
        c1.z = pack_h2(x[12] * scale, x[13] * scale); c1.w = pack_h2(x[14] * scale, x[15] * scale);
        // B tile of heads 4g..4g+3 ([32 rows x 64 k], K-major, 128-byte swizzle): head h at k = 16 (h & 3) .. +15;
        // row n = r < 16 holds S_h[.][r], row 16 holds z_h
        const uint32_t tile = sbase + OFF_B + bb.slot * B_BUF + (h >> 2) * 4096;
        const int lc = 2 * (h & 3);                       // first logical 16-byte chunk of the head
        sts128(tile + r * 128 + ((lc ^ (r & 7)) << 4), c0);
        sts128(tile + r * 128 + (((lc + 1) ^ (r & 7)) << 4), c1);
        sts16(tile + 16 * 128 + ((lc + (r >> 3)) << 4) + (r & 7) * 2, __half_as_ushort(__float2half_rn(zv * scale)));
        proxy_fence();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(smem_u32(&ctrl.b_full[bb.slot]));
        advance<NB>(bb);
      } else {
        // piece of a long window: partial state -> workspace slot of the window (fp32 atomics)
        float* slot = ws + kWsHeaderFloats + ((size_t)(d.w / (kFuseMax + 1)) * H + (h0 + h)) * (size_t)((D + 1) * D);
#pragma unroll
        for (int p = 0; p < 16; ++p) atomicAdd(slot + p * D + r, x[p]);
        atomicAdd(slot + D * D + r, zv);
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive_n(smem_u32(&ctrl.region_free[rg.slot]), NEPI / NCONV);
      }
      advance<NSL>(rg);
    }
  } else {
    // =========================== epilogue: one thread per output row ===========================
    const int ew = warp - WARP_EPI0;
    const int quad = warp & 3;                           // TMEM lane quadrant of this warp
    Cur it{0, 0}, rg{0, 0};
    TileRing<NQT> qr{0, 0u};
    uint32_t of_ph = 0;                                  // parity of the next o_full completion, per region
    while (true) {
      const int4 d = next_item(it);
      if (d.x == IT_END) break;
      if (d.x == IT_PACK) { qr.alloc(1); continue; }
      if (d.x == IT_PIECE) { advance<NSL>(rg); continue; }
      const int s = d.y, m = d.z;
      const int T16 = (m + 15) >> 4;
      const uint32_t region = tmem + (uint32_t)(rg.slot * REGION_COLS);
      for (int b = 0; b * 8 < T16; ++b) {
        const int first = qr.alloc(min(8, T16 - 8 * b));
        const int rows = min(128, m - 128 * b);          // valid rows of this block
        mbar_wait_wd(smem_u32(&ctrl.o_full[rg.slot]), (of_ph >> rg.slot) & 1u);
        of_ph ^= 1u << rg.slot;
        tc_fence_after();
        if (32 * quad < rows) {
#pragma unroll 1
         for (int hf = 0; hf < EPI_HALVES; ++hf) {
          const int half = EPI_HALVES == 2 ? hf : (ew >> 2);   // which 4 heads (64 channels)
          const uint32_t stage0 = sbase + OFF_Q + half * Q_REG;   // staging: this half of the (now dead) Q tiles
          const uint32_t taddr = region + ((uint32_t)(32 * quad) << 16) + 128 * half;
          const int rib = 32 * quad + lane;              // row of the block this thread owns
          const uint32_t srow = stage0 + (first + (rib >> 4)) * 2048 + (rib & 15) * 128;
#pragma unroll
          for (int hp = 0; hp < 2; ++hp) {               // two heads at a time
            uint32_t va[16], vb[16], da, db;
            tmem_ld16(taddr + 64 * hp, va);
            tmem_ld1(taddr + 64 * hp + 16, da);
            tmem_ld16(taddr + 64 * hp + 32, vb);
            tmem_ld1(taddr + 64 * hp + 48, db);
            tmem_wait_ld();
            const float ia = fast_rcp(__uint_as_float(da)), ib = fast_rcp(__uint_as_float(db));
            uint4 o[4];
#pragma unroll
            for (int c = 0; c < 2; ++c) {
              o[c].x = pack_out<BF16>(__uint_as_float(va[8 * c + 0]) * ia, __uint_as_float(va[8 * c + 1]) * ia);
              o[c].y = pack_out<BF16>(__uint_as_float(va[8 * c + 2]) * ia, __uint_as_float(va[8 * c + 3]) * ia);
              o[c].z = pack_out<BF16>(__uint_as_float(va[8 * c + 4]) * ia, __uint_as_float(va[8 * c + 5]) * ia);
              o[c].w = pack_out<BF16>(__uint_as_float(va[8 * c + 6]) * ia, __uint_as_float(va[8 * c + 7]) * ia);
              o[2 + c].x = pack_out<BF16>(__uint_as_float(vb[8 * c + 0]) * ib, __uint_as_float(vb[8 * c + 1]) * ib);
              o[2 + c].y = pack_out<BF16>(__uint_as_float(vb[8 * c + 2]) * ib, __uint_as_float(vb[8 * c + 3]) * ib);
              o[2 + c].z = pack_out<BF16>(__uint_as_float(vb[8 * c + 4]) * ib, __uint_as_float(vb[8 * c + 5]) * ib);
              o[2 + c].w = pack_out<BF16>(__uint_as_float(vb[8 * c + 6]) * ib, __uint_as_float(vb[8 * c + 7]) * ib);
            }
            if (rib < rows) {
#pragma unroll
              for (int c = 0; c < 4; ++c) sts128(srow + (((4 * hp + c) ^ (rib & 7)) << 4), o[c]);
            }
          }
          __syncwarp();
          // coalesced copy-out: per instruction 4 rows x 128 bytes (lane -> row 4 it + lane/8, chunk lane%8)
          const int nr = min(32, rows - 32 * quad);
          T* obase = out + (size_t)(s + 128 * b + 32 * quad) * Ctot + col0 + 64 * half + (lane & 7) * 8;
          uint4 x[8];
#pragma unroll
          for (int i = 0; i < 8; ++i) {
            const int row = 4 * i + (lane >> 3), rb = 32 * quad + row;
            if (row < nr)
              x[i] = lds128(stage0 + (first + (rb >> 4)) * 2048 + (rb & 15) * 128 + (((lane & 7) ^ (rb & 7)) << 4));
          }
#pragma unroll
          for (int i = 0; i < 8; ++i) {
            const int row = 4 * i + (lane >> 3);
            if (row < nr) *reinterpret_cast<uint4*>(obase + (size_t)row * Ctot) = x[i];
          }
         }
          proxy_fence();
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) {
          // relaxed: what these arrivals publish (TMEM reads, shared-memory reads of the staging tiles) is complete;
          // a releasing arrive would also wait for the global stores above to be acknowledged
          mbar_arrive_relaxed(smem_u32(&ctrl.q_empty[first]));
          mbar_arrive_relaxed(smem_u32((b + 1) * 8 < T16 ? &ctrl.o_drained[rg.slot] : &ctrl.region_free[rg.slot]));
        }
      }
      advance<NSL>(rg);
    }
  }

  // ---- teardown ---------------------------------------------------------------------------------------
  tc_fence_before();
  __syncthreads();
  if (warp == WARP_SMMA) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(TMEM_COLS));
  }
}

template <bool BF16, typename T>
cudaError_t umma_launch(const Problem& p, cudaStream_t st) {
  Maps maps;
  const int Ctot = p.H * D;
  const void* base[3] = {p.q, p.k, p.v};
  for (int t = 0; t < 3; ++t)
    for (int k = 0; k < 4; ++k)
      if (!make_map(&maps.m[t][k], base[t], p.N, Ctot, 16 << k)) return cudaErrorInvalidValue;
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
  return cudaLaunchKernelEx(&cfg, kern, maps, (const T*)p.q, (const T*)p.k, (const T*)p.v, p.off, (T*)p.out,
                            p.ws_state, p.N, p.W, p.H, span);
}

}  // namespace


bool forward_umma_supported(const Problem& p, int dt) {
  if (dt != SLA_F16 || p.phi != SLA_PHI_ELU1) return false;
  if (p.d != D || (p.H * p.d) % 128 != 0) return false;
  return encode_fn() != nullptr;
}

cudaError_t launch_forward_umma_main(const Problem& p, int dt, cudaStream_t st) {
  (void)dt;
  cudaError_t e = umma_launch<false, __half>(p, st);
  return e;
}

}  // namespace sla
