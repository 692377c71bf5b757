// sla_fwd_tc.cu -- SLA forward for fp16 / bf16 I/O on sm_100a: TMA-streamed, warp-per-head,
// tensor-core (mma.sync m16n8k16, fp32 accumulate) contractions, window state kept in registers.
//
// Design:
//   * The flat window-sorted matrix is cut into equal row spans, one per CTA
//     (load balance by rows/chunks, not by window -- PAPER.md:93 Fig. 3a).  A CTA owns every window
//     of <= FUSE_MAX rows whose middle row lies in its span (processed whole, state never leaves the
//     SM) and, for longer windows, the piece that intersects its span (partial state -> fp32
//     atomics into the workspace; outputs by a second launch of this kernel in OUTPASS mode).
//   * Memory streaming is decoupled from the window structure: two producer lanes stream the CTA's
//     rows of K,V and of Q through two shared-memory rings with 2-D TMA (128-byte swizzle) and
//     mbarriers, regardless of where windows begin and end.
//   * Consumer warp h owns head h of the slab (8 heads).  Per 16-row tile it forms
//       S^T += V^T phi(K)   (Eq. 3 numerator state; contraction over voxels)
//       z   += 1^T phi(K)   (normaliser)
//     with ldmatrix.trans operands, then per 16-row Q tile  O = phi(Q) S / (phi(Q) z).
//     The accumulator fragment of S^T is exactly the B fragment of S for the output mma.
//   * Precision: operands are fp16, accumulation fp32.  Windows of <= 16 rows are packed into 16-row
//     tiles and evaluated in the quadratic form with phi() in fp32 and split operands (x = hi + lo,
//     both fp16: ~22-bit products); longer windows use phi() in fp16x2, one term, and the state scaled
//     by the power of two that brings its largest z into [1, 2) (the ratio of Eq. 3 is scale invariant).
#include <cuda.h>

#include <atomic>

#include "sla_internal.cuh"

namespace sla {
namespace {

constexpr int NW = 8;                       // consumer warps = heads per slab
#ifndef SLA_HPW
#define SLA_HPW 1
#endif
#ifndef SLA_MINB
#define SLA_MINB 3
#endif
#ifndef SLA_NST
#define SLA_NST 3
#endif
#ifndef SLA_SR
#define SLA_SR 32
#endif
constexpr int NST = SLA_NST;                // ring stages per stream at d_h = 16 (and the size of the barrier arrays)
constexpr int QUAD_MAX = 16;                // windows up to this length are packed into quadratic-form tiles
constexpr int kSpanTableMagic = 0x534c4154; // "SLAT": first word of a span table (sla_build_span_table)

template <int D> struct Cfg {
  static constexpr int SR = SLA_SR;                       // rows per ring stage
  static constexpr int NBOX = NW * D / 64;                // 128-byte column boxes per slab row
  static constexpr int BOX_BYTES = SR * 128;
  static constexpr int T_STAGE = NBOX * BOX_BYTES;        // bytes of one tensor's stage (4 / 8 KB)
  static constexpr int KV_STAGE = 2 * T_STAGE;
  // d_h = 32: a stage is twice as large; two stages instead of three let two CTAs share an SM (config 2: 188 -> 147 us)
  static constexpr int NSTG = (D == 32 && NST > 2) ? 2 : NST;
  static constexpr int RING_BYTES = NSTG * (KV_STAGE + T_STAGE);
  static constexpr int SMEM_DYN = RING_BYTES + 1024;      // + alignment slack (swizzle needs 1 KB)
  static constexpr int HPW = (D == 16) ? SLA_HPW : 1;     // heads per consumer warp (ILP, shared bookkeeping)
  static constexpr int NCW = NW / HPW;                    // consumer warps per CTA
  static constexpr int THREADS = (NCW + 1) * 32;          // + one producer warp
};

#include "sla_tc_common.cuh"

// ---- state of one (window, head) in mma fragments --------------------------------------------------
//   ST[mt][nt][c]: S^T[r][p], r = 16*mt + g + 8*(c/2), p = 8*nt + 2*t + (c%2)   (g = lane/4, t = lane%4)
//   Z[nt][c]     : z[p], p = 8*nt + 2*t + (c%2)  (same value in every row)
template <int D> struct State {
  float ST[D / 16][D / 8][4];
  float Z[D / 8][4];
  __device__ __forceinline__ void clear() {
#pragma unroll
    for (int a = 0; a < D / 16; ++a)
#pragma unroll
      for (int b = 0; b < D / 8; ++b)
#pragma unroll
        for (int c = 0; c < 4; ++c) ST[a][b][c] = 0.f;
#pragma unroll
    for (int b = 0; b < D / 8; ++b)
#pragma unroll
      for (int c = 0; c < 4; ++c) Z[b][c] = 0.f;
  }
};

// One 16-row K/V tile starting at relative row `rel0` with `nvalid` rows of the current window.
//
// Shared addresses: the head's 16-byte chunks are hl*(D/8) + 2*cp + csel, all inside one 128-byte box
// row, and chunk bit 1 = cp, so under the 128-byte swizzle (chunk ^ (row & 7)) the address of column
// pair cp is the address of pair 0 with bit 5 flipped.  `a0` is that pair-0 address of this lane's
// ldmatrix row in the K stage (V: + T_STAGE); full 32-row steps pass it in and advance it by one ring
// slot per step instead of recomputing stage, slot and swizzle (process_window).
template <int D>
__device__ __forceinline__ uint32_t lane_tile_addr(const RingView& rv, int slot_bytes, int hl, int rel0, int nvalid) {
  const int lane = threadIdx.x & 31;
  const int mi = lane >> 3;
  int trow = (lane & 7) + 8 * (mi >> 1);           // tile row this lane addresses for ldmatrix
  if (trow >= nvalid) trow = 0;                    // clamp: row 0 of the tile is always valid
  return ring_addr<D>(rv, slot_bytes, 0, rel0 + trow, hl * (D / 8) + (mi & 1));
}
// advance a lane address by one ring slot (the next stage), wrapping at the end of the ring
__device__ __forceinline__ uint32_t ring_next_slot(uint32_t a, uint32_t ring_end, int slot_bytes, int nst) {
  a += (uint32_t)slot_bytes;
  return a >= ring_end ? a - (uint32_t)(nst * slot_bytes) : a;
}

template <int D, int MODE, bool PRECISE, bool FULL = false>
__device__ __forceinline__ void kv_tile(const RingView& rv, int hl, int rel0, int nvalid_in, State<D>& s,
                                        uint32_t a0_in = 0u) {
  constexpr bool BF16 = (MODE & 1) != 0;   // I/O dtype bf16
  constexpr int PHI = MODE >> 1;            // feature map (sla_feature_map_t)
  (void)BF16; (void)PHI;
  const int nvalid = FULL ? 16 : nvalid_in;
  using C = Cfg<D>;
  const int lane = threadIdx.x & 31;
  const int t = lane & 3;
  const uint32_t a0 = FULL ? a0_in : lane_tile_addr<D>(rv, C::KV_STAGE, hl, rel0, nvalid);
  const uint32_t ones = 0x3C003C00u;               // fp16 {1,1}
#pragma unroll
  for (int cp = 0; cp < D / 16; ++cp) {            // 16-channel column pairs of the head
    uint32_t kr[4], vr[4];
    ldsm_x4_t(a0 ^ (uint32_t)(cp << 5), kr);
    ldsm_x4_t((a0 ^ (uint32_t)(cp << 5)) + C::T_STAGE, vr);
    // phi(K) fragments: kr[0],kr[1] hold voxels j = 2t,2t+1; kr[2],kr[3] hold j = 2t+8,2t+9
    uint32_t bhi[4], blo[4];
    if (PRECISE) {
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const int j0 = 2 * t + 8 * (i >> 1);
        float2 x = unpack2<BF16>(kr[i]);
        float b0 = (j0 < nvalid) ? phi_fast<PHI>(x.x) : 0.f;
        float b1 = (j0 + 1 < nvalid) ? phi_fast<PHI>(x.y) : 0.f;
        split_h2(b0, b1, bhi[i], blo[i]);
      }
    } else {
#pragma unroll
      for (int i = 0; i < 4; ++i) { bhi[i] = phi_h2<BF16, PHI>(kr[i]); blo[i] = 0u; }
      if (nvalid < 16) {                            // ragged last tile of the window: zero phi(K) rows
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          const int j0 = 2 * t + 8 * (i >> 1);
          const uint32_t msk = ((j0 < nvalid) ? 0x0000FFFFu : 0u) | ((j0 + 1 < nvalid) ? 0xFFFF0000u : 0u);
          bhi[i] &= msk;
        }
      }
    }
    if (BF16) {                                     // V: bf16 -> fp16 (exact in the normal range)
#pragma unroll
      for (int i = 0; i < 4; ++i) { float2 x = unpack2<true>(vr[i]); vr[i] = pack_h2(x.x, x.y); }
    }
    // K fragment registers: n-tile 2cp   -> (b0,b1) = (r0,r2);  n-tile 2cp+1 -> (r1,r3)
    // V fragment registers: m-tile cp    -> (a0,a1,a2,a3) = (r0,r1,r2,r3)
#pragma unroll
    for (int half = 0; half < 2; ++half) {
      const int nt = 2 * cp + half;
      const uint32_t b0 = bhi[half], b1 = bhi[2 + half];
      mma16816(s.Z[nt], ones, ones, ones, ones, b0, b1);
      if (PRECISE) mma16816(s.Z[nt], ones, ones, ones, ones, blo[half], blo[2 + half]);
    }
    // every m-tile of V^T meets every n-tile of phi(K): keep V fragments of all column pairs
    // (D=16: one pair; D=32: handled by the second pass below)
    if (D == 16) {
#pragma unroll
      for (int half = 0; half < 2; ++half) {
        mma16816(s.ST[0][half], vr[0], vr[1], vr[2], vr[3], bhi[half], bhi[2 + half]);
        if (PRECISE) mma16816(s.ST[0][half], vr[0], vr[1], vr[2], vr[3], blo[half], blo[2 + half]);
      }
    } else {
      // D == 32: load both V column pairs for this K column pair
#pragma unroll
      for (int mt = 0; mt < D / 16; ++mt) {
        uint32_t va[4];
        if (mt == cp) { va[0] = vr[0]; va[1] = vr[1]; va[2] = vr[2]; va[3] = vr[3]; }
        else {
          ldsm_x4_t((a0 ^ (uint32_t)(mt << 5)) + C::T_STAGE, va);
          if (BF16) {
#pragma unroll
            for (int i = 0; i < 4; ++i) { float2 x = unpack2<true>(va[i]); va[i] = pack_h2(x.x, x.y); }
          }
        }
#pragma unroll
        for (int half = 0; half < 2; ++half) {
          const int nt = 2 * cp + half;
          mma16816(s.ST[mt][nt], va[0], va[1], va[2], va[3], bhi[half], bhi[2 + half]);
          if (PRECISE) mma16816(s.ST[mt][nt], va[0], va[1], va[2], va[3], blo[half], blo[2 + half]);
        }
      }
    }
  }
}

// B operands of the output mma, built once per (window, head) from the state.
//   B[n2][ks] covers output channels r = 8*n2 .. 8*n2+7 and contraction p = 16*ks .. 16*ks+15.
template <int D> struct OutOperands {
  uint32_t hi[D / 8][D / 16][2], lo[D / 8][D / 16][2];
  uint32_t zhi[D / 16][2], zlo[D / 16][2];
  float eps;   // epsilon of the denominator on the scale of the operands (eps * scale)
};

// the factor applied to a state before its fp16 rounding: z_scale (sla_tc_base.cuh)
template <int D>
__device__ __forceinline__ float state_scale(const State<D>& s) { return z_scale<D / 8>(s.Z); }

template <int D, bool PRECISE>
__device__ __forceinline__ void make_out_operands(const State<D>& s, float scale, float eps, OutOperands<D>& o) {
  o.eps = eps * scale;
#pragma unroll
  for (int n2 = 0; n2 < D / 8; ++n2)
#pragma unroll
    for (int ks = 0; ks < D / 16; ++ks)
#pragma unroll
      for (int b = 0; b < 2; ++b) {
        const float x0 = s.ST[n2 / 2][2 * ks + b][2 * (n2 & 1)] * scale;
        const float x1 = s.ST[n2 / 2][2 * ks + b][2 * (n2 & 1) + 1] * scale;
        if (PRECISE) split_h2(x0, x1, o.hi[n2][ks][b], o.lo[n2][ks][b]);
        else { o.hi[n2][ks][b] = pack_h2(x0, x1); o.lo[n2][ks][b] = 0u; }
      }
#pragma unroll
  for (int ks = 0; ks < D / 16; ++ks)
#pragma unroll
    for (int b = 0; b < 2; ++b) {
      const float x0 = s.Z[2 * ks + b][0] * scale, x1 = s.Z[2 * ks + b][1] * scale;
      if (PRECISE) split_h2(x0, x1, o.zhi[ks][b], o.zlo[ks][b]);
      else { o.zhi[ks][b] = pack_h2(x0, x1); o.zlo[ks][b] = 0u; }
    }
}

// One 16-row Q tile: out rows [row0, row0+nvalid) of head h.  `lane_out` = this lane's first output
// element (row0 + g, head column + 2t); `o8` = 8 rows in elements.
template <int D, int MODE, bool PRECISE, typename T, bool FULL = false>
__device__ __forceinline__ void q_tile(const RingView& rv, int hl, int rel0, int nvalid_in,
                                       const OutOperands<D>& o, T* __restrict__ lane_out, size_t o8,
                                       uint32_t a0_in = 0u) {
  constexpr bool BF16 = (MODE & 1) != 0;   // I/O dtype bf16
  constexpr int PHI = MODE >> 1;            // feature map (sla_feature_map_t)
  (void)BF16; (void)PHI;
  const int nvalid = FULL ? 16 : nvalid_in;
  using C = Cfg<D>;
  const int lane = threadIdx.x & 31;
  const int g = lane >> 2;
  const uint32_t a0 = FULL ? a0_in : lane_tile_addr<D>(rv, C::T_STAGE, hl, rel0, nvalid);
  uint32_t ahi[D / 16][4], alo[D / 16][4];
#pragma unroll
  for (int ks = 0; ks < D / 16; ++ks) {
    uint32_t qr[4];
    ldsm_x4(a0 ^ (uint32_t)(ks << 5), qr);
    // registers (rows0-7,c0),(rows0-7,c1),(rows8-15,c0),(rows8-15,c1) -> a0=r0, a1=r2, a2=r1, a3=r3
    const int perm[4] = {0, 2, 1, 3};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      if (PRECISE) {
        float2 x = unpack2<BF16>(qr[perm[i]]);
        split_h2(phi_fast<PHI>(x.x), phi_fast<PHI>(x.y), ahi[ks][i], alo[ks][i]);
      } else {
        ahi[ks][i] = phi_h2<BF16, PHI>(qr[perm[i]]);
        alo[ks][i] = 0u;
      }
    }
  }
  float den[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
  for (int ks = 0; ks < D / 16; ++ks) {
    mma16816(den, ahi[ks][0], ahi[ks][1], ahi[ks][2], ahi[ks][3], o.zhi[ks][0], o.zhi[ks][1]);
    if (PRECISE) {
      mma16816(den, alo[ks][0], alo[ks][1], alo[ks][2], alo[ks][3], o.zhi[ks][0], o.zhi[ks][1]);
      mma16816(den, ahi[ks][0], ahi[ks][1], ahi[ks][2], ahi[ks][3], o.zlo[ks][0], o.zlo[ks][1]);
    }
  }
  const float inv0 = fast_rcp(den[0] + o.eps), inv1 = fast_rcp(den[2] + o.eps);
#pragma unroll
  for (int n2 = 0; n2 < D / 8; ++n2) {
    float acc[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
    for (int ks = 0; ks < D / 16; ++ks) {
      mma16816(acc, ahi[ks][0], ahi[ks][1], ahi[ks][2], ahi[ks][3], o.hi[n2][ks][0], o.hi[n2][ks][1]);
      if (PRECISE) {
        mma16816(acc, alo[ks][0], alo[ks][1], alo[ks][2], alo[ks][3], o.hi[n2][ks][0], o.hi[n2][ks][1]);
        mma16816(acc, ahi[ks][0], ahi[ks][1], ahi[ks][2], ahi[ks][3], o.lo[n2][ks][0], o.lo[n2][ks][1]);
      }
    }
    uint32_t* p0 = reinterpret_cast<uint32_t*>(lane_out + 8 * n2);
    uint32_t* p1 = reinterpret_cast<uint32_t*>(lane_out + o8 + 8 * n2);
    if (FULL || g < nvalid) *p0 = pack_out<BF16>(acc[0] * inv0, acc[1] * inv0);
    if (FULL || g + 8 < nvalid) *p1 = pack_out<BF16>(acc[2] * inv1, acc[3] * inv1);
  }
}

// packed short windows (quad_tile_core, sla_tc_base.cuh) on rows rel0.. of this CTA's K/V and Q rings
template <int D, int MODE, typename T>
__device__ __forceinline__ void quad_tile(const RingView& kv, const RingView& qv, int hl, int rel0,
                                          int nvalid, int wid, T* __restrict__ out_rows, int C_total, float eps) {
  constexpr bool BF16 = (MODE & 1) != 0;   // I/O dtype bf16
  constexpr int PHI = MODE >> 1;            // feature map (sla_feature_map_t)
  (void)BF16; (void)PHI;
  using C = Cfg<D>;
  quad_tile_core<D, BF16, T, PHI>(
      [&](int r, int c) { return ring_addr<D>(qv, C::T_STAGE, 0, rel0 + r, c); },
      [&](int r, int c) { return ring_addr<D>(kv, C::KV_STAGE, 0, rel0 + r, c); },
      [&](int r, int c) { return ring_addr<D>(kv, C::KV_STAGE, C::T_STAGE, rel0 + r, c); }, hl, nvalid, wid,
      out_rows, C_total, eps);
}

// ---- CTA-level shared control block ----------------------------------------------------------------
struct Ctrl {
  unsigned long long full_kv[NST], empty_kv[NST], full_q[NST], empty_q[NST];
  int wa;            // window containing row R0
  int stream_begin;  // S0: first row any owned item touches
  int stream_end;    // one past the last row any owned item touches (>= S0)
};

// One whole (fused) window [s,e) for head slot hl: state pass over K,V then output pass over Q.
// Rows are addressed relative to S0, the first row of this CTA's streams.  Two 16-row tiles per
// iteration: one wait/release bookkeeping step per 32 rows and two independent dependency chains.
template <int D, int MODE, bool PRECISE, typename T>
__device__ __forceinline__ void process_window(RingView& kv, RingView& qv, int hl, int nh, int S0, int s,
                                               int e, T* __restrict__ out_head /*out + head column*/,
                                               int Ctot, float eps) {
  constexpr bool BF16 = (MODE & 1) != 0;   // I/O dtype bf16
  constexpr int PHI = MODE >> 1;            // feature map (sla_feature_map_t)
  (void)BF16; (void)PHI;
  using C = Cfg<D>;
  State<D> st[C::HPW];
#pragma unroll
  for (int j = 0; j < C::HPW; ++j) st[j].clear();
  const int lane = threadIdx.x & 31;
  // Lane addresses of the two 16-row tiles of a full 32-row step: computed once per pass, then moved
  // to the next ring slot each step (a step is exactly one stage of rows).
  uint32_t ak[C::HPW][2];
  ring_release_below<C::SR>(kv, s - S0);   // ring_addr needs the stage within NST of `released`
#pragma unroll
  for (int j = 0; j < C::HPW; ++j) {
    ak[j][0] = lane_tile_addr<D>(kv, C::KV_STAGE, hl + j, s - S0, 16);
    ak[j][1] = lane_tile_addr<D>(kv, C::KV_STAGE, hl + j, s - S0 + 16, 16);
  }
  const uint32_t kv_end = kv.base + C::NSTG * C::KV_STAGE;
  for (int r = s; r < e; r += 32) {
    const int nv = min(32, e - r), rel = r - S0;
    // stages entirely below this step go back to the producer first: a wait must never pin older
    // stages.  The first step's were released above; every later step frees exactly one (SR = 32).
    if (C::SR != 32) ring_release_below<C::SR>(kv, rel);
    else if (r != s) ring_release_one(kv);
    ring_wait_upto(kv, (rel + nv - 1) / C::SR);
#pragma unroll
    for (int j = 0; j < C::HPW; ++j)
      if (j < nh) {
        if (nv == 32) {   // two full tiles, one basic block: the two dependency chains interleave
          kv_tile<D, MODE, PRECISE, true>(kv, hl + j, rel, 16, st[j], ak[j][0]);
          kv_tile<D, MODE, PRECISE, true>(kv, hl + j, rel + 16, 16, st[j], ak[j][1]);
          ak[j][0] = ring_next_slot(ak[j][0], kv_end, C::KV_STAGE, C::NSTG);
          ak[j][1] = ring_next_slot(ak[j][1], kv_end, C::KV_STAGE, C::NSTG);
        } else {
          kv_tile<D, MODE, PRECISE>(kv, hl + j, rel, min(16, nv), st[j]);
          if (nv > 16) kv_tile<D, MODE, PRECISE>(kv, hl + j, rel + 16, nv - 16, st[j]);
        }
      }
  }
  OutOperands<D> oo[C::HPW];
#pragma unroll
  for (int j = 0; j < C::HPW; ++j) make_out_operands<D, PRECISE>(st[j], state_scale<D>(st[j]), eps, oo[j]);
  uint32_t aq[C::HPW][2];
  ring_release_below<C::SR>(qv, s - S0);
#pragma unroll
  for (int j = 0; j < C::HPW; ++j) {
    aq[j][0] = lane_tile_addr<D>(qv, C::T_STAGE, hl + j, s - S0, 16);
    aq[j][1] = lane_tile_addr<D>(qv, C::T_STAGE, hl + j, s - S0 + 16, 16);
  }
  const uint32_t q_end = qv.base + C::NSTG * C::T_STAGE;
  const size_t o8 = (size_t)8 * Ctot;
  // this lane's first output element: row s + g, head column + 2t; 32 rows further every step
  T* lp = out_head + (size_t)(s + (lane >> 2)) * Ctot + 2 * (lane & 3);
  for (int r = s; r < e; r += 32, lp += 4 * o8) {
    const int nv = min(32, e - r), rel = r - S0;
    if (C::SR != 32) ring_release_below<C::SR>(qv, rel);
    else if (r != s) ring_release_one(qv);
    ring_wait_upto(qv, (rel + nv - 1) / C::SR);
#pragma unroll
    for (int j = 0; j < C::HPW; ++j)
      if (j < nh) {
        T* oh = lp + j * D;
        if (nv == 32) {
          q_tile<D, MODE, PRECISE, T, true>(qv, hl + j, rel, 16, oo[j], oh, o8, aq[j][0]);
          q_tile<D, MODE, PRECISE, T, true>(qv, hl + j, rel + 16, 16, oo[j], oh + 2 * o8, o8, aq[j][1]);
          aq[j][0] = ring_next_slot(aq[j][0], q_end, C::T_STAGE, C::NSTG);
          aq[j][1] = ring_next_slot(aq[j][1], q_end, C::T_STAGE, C::NSTG);
        } else {
          q_tile<D, MODE, PRECISE, T>(qv, hl + j, rel, min(16, nv), oo[j], oh, o8);
          if (nv > 16) q_tile<D, MODE, PRECISE, T>(qv, hl + j, rel + 16, nv - 16, oo[j], oh + 2 * o8, o8);
        }
      }
  }
}

// The piece [ps,pe) of a split window: partial state -> workspace atomics.
template <int D, int MODE>
__device__ __forceinline__ void process_piece(RingView& kv, int hl, int nh, int S0, int ps, int pe,
                                              float* __restrict__ slot /*slot of head hl*/) {
  constexpr bool BF16 = (MODE & 1) != 0;   // I/O dtype bf16
  constexpr int PHI = MODE >> 1;            // feature map (sla_feature_map_t)
  (void)BF16; (void)PHI;
  using C = Cfg<D>;
  const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
  State<D> st[C::HPW];
#pragma unroll
  for (int j = 0; j < C::HPW; ++j) st[j].clear();
  for (int r = ps; r < pe; r += 32) {
    const int nv = min(32, pe - r), rel = r - S0;
    ring_release_below<C::SR>(kv, rel);
    ring_wait_upto(kv, (rel + nv - 1) / C::SR);
#pragma unroll
    for (int j = 0; j < C::HPW; ++j)
      if (j < nh) {
        kv_tile<D, MODE, false>(kv, hl + j, rel, min(16, nv), st[j]);
        if (nv > 16) kv_tile<D, MODE, false>(kv, hl + j, rel + 16, nv - 16, st[j]);
      }
  }
#pragma unroll
  for (int j = 0; j < C::HPW; ++j)
    if (j < nh) {
      float* sl = slot + j * (D + 1) * D;
#pragma unroll
      for (int mt = 0; mt < D / 16; ++mt)
#pragma unroll
        for (int nt = 0; nt < D / 8; ++nt)
#pragma unroll
          for (int c = 0; c < 4; ++c) {
            const int r = 16 * mt + g + 8 * (c >> 1), p = 8 * nt + 2 * t + (c & 1);
            atomicAdd(sl + p * D + r, st[j].ST[mt][nt][c]);
          }
      if (g == 0) {
#pragma unroll
        for (int nt = 0; nt < D / 8; ++nt)
#pragma unroll
          for (int c = 0; c < 2; ++c) atomicAdd(sl + D * D + 8 * nt + 2 * t + c, st[j].Z[nt][c]);
      }
    }
}

// Output pass for the piece [ps,pe) of a split window of m rows: the complete state is read from the
// workspace slot (fp32 [d+1, d]: rows 0..d-1 = S, row d = z) into the mma fragment layout.
template <int D, int MODE, typename T>
__device__ __forceinline__ void output_piece(RingView& qv, int hl, int S0, int ps, int pe, int m,
                                             const float* __restrict__ slot, T* __restrict__ out_head,
                                             int Ctot, float eps) {
  constexpr bool BF16 = (MODE & 1) != 0;   // I/O dtype bf16
  constexpr int PHI = MODE >> 1;            // feature map (sla_feature_map_t)
  (void)BF16; (void)PHI;
  using C = Cfg<D>;
  const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
  State<D> st;
#pragma unroll
  for (int mt = 0; mt < D / 16; ++mt)
#pragma unroll
    for (int nt = 0; nt < D / 8; ++nt)
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        const int r = 16 * mt + g + 8 * (c >> 1), p = 8 * nt + 2 * t + (c & 1);
        st.ST[mt][nt][c] = slot[p * D + r];
      }
#pragma unroll
  for (int nt = 0; nt < D / 8; ++nt)
#pragma unroll
    for (int c = 0; c < 4; ++c) st.Z[nt][c] = slot[D * D + 8 * nt + 2 * t + (c & 1)];
  (void)m;
  OutOperands<D> oo;
  make_out_operands<D, false>(st, state_scale<D>(st), eps, oo);
  uint32_t aq[2];
  ring_release_below<C::SR>(qv, ps - S0);
  aq[0] = lane_tile_addr<D>(qv, C::T_STAGE, hl, ps - S0, 16);
  aq[1] = lane_tile_addr<D>(qv, C::T_STAGE, hl, ps - S0 + 16, 16);
  const uint32_t q_end = qv.base + C::NSTG * C::T_STAGE;
  const size_t o8 = (size_t)8 * Ctot;
  T* lp = out_head + (size_t)(ps + g) * Ctot + 2 * t;
  for (int r = ps; r < pe; r += 32, lp += 4 * o8) {
    const int nv = min(32, pe - r), rel = r - S0;
    if (C::SR != 32) ring_release_below<C::SR>(qv, rel);
    else if (r != ps) ring_release_one(qv);
    ring_wait_upto(qv, (rel + nv - 1) / C::SR);
    if (nv == 32) {
      q_tile<D, MODE, false, T, true>(qv, hl, rel, 16, oo, lp, o8, aq[0]);
      q_tile<D, MODE, false, T, true>(qv, hl, rel + 16, 16, oo, lp + 2 * o8, o8, aq[1]);
      aq[0] = ring_next_slot(aq[0], q_end, C::T_STAGE, C::NSTG);
      aq[1] = ring_next_slot(aq[1], q_end, C::T_STAGE, C::NSTG);
    } else {
      q_tile<D, MODE, false, T>(qv, hl, rel, min(16, nv), oo, lp, o8);
      if (nv > 16) q_tile<D, MODE, false, T>(qv, hl, rel + 16, nv - 16, oo, lp + 2 * o8, o8);
    }
  }
}

// OUTPASS = false: the main kernel.  OUTPASS = true: the second pass of the general entry -- outputs of
// the pieces of windows longer than kFuseMax, whose complete states the main kernel left in the
// workspace; it streams only Q and exits at once if the main kernel met no such window.
template <int D, int MODE, typename T, bool OUTPASS>
__global__ void __launch_bounds__(Cfg<D>::THREADS, (D == 16 ? SLA_MINB : 2))
sla_fwd_tc_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmK,
                  const __grid_constant__ CUtensorMap tmV, const int32_t* __restrict__ off,
                  T* __restrict__ out, float* __restrict__ ws, int N, int W, int H, int span, float eps,
                  const int4* __restrict__ table) {
  using C = Cfg<D>;
  extern __shared__ uint8_t dyn_smem[];
  __shared__ Ctrl ctrl;
  // Programmatic dependent launch (the host side opts in with the stream-serialisation attribute): this
  // grid may become resident while the previous kernel of the stream is still in its tail.  Nothing that
  // kernel may have written (offsets, tensors, workspace) is touched before griddepcontrol.wait, which
  // returns once that whole grid has completed; only the barrier set-up runs ahead.  The next kernel is
  // released at once: it can only become resident when every CTA of this grid has started.
  asm volatile("griddepcontrol.launch_dependents;");
  if (OUTPASS) {
    asm volatile("griddepcontrol.wait;" ::: "memory");
    if (reinterpret_cast<const volatile int*>(ws)[0] == 0) return;   // no split window in this call
  }
  const uint32_t ring = (smem_u32(dyn_smem) + 1023u) & ~1023u;
  const uint32_t kv_base = ring, q_base = ring + C::NSTG * C::KV_STAGE;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  // CTAs are dispatched in blockIdx order and the grid runs in several waves (spans are short).
  // Map CTAs to spans outside-in: both ends of the row-major window order first.  In a LiDAR scene
  // those are the far-range rows: sparse, many 1-4 voxel windows, the slowest spans per row (measured
  // 6 rows/us against 11-12 for dense spans), so they get the head start and the fast dense spans of
  // the middle fill the tail.
  const int nspan = gridDim.x;
  const int bx = blockIdx.x;
  const int sidx = (bx & 1) ? nspan - 1 - (bx >> 1) : (bx >> 1);
  const int R0 = sidx * span, R1 = min(R0 + span, N);
  const int h0 = blockIdx.y * NW;
  const int nheads = min(NW, H - h0);                       // heads of this slab
  const int nact = (nheads + C::HPW - 1) / C::HPW;           // active consumer warps
  const int Ctot = H * D;

  if (threadIdx.x == 0) {
    for (int i = 0; i < C::NSTG; ++i) {
      mbar_init(smem_u32(&ctrl.full_kv[i]), 1);
      mbar_init(smem_u32(&ctrl.empty_kv[i]), nact);
      mbar_init(smem_u32(&ctrl.full_q[i]), 1);
      mbar_init(smem_u32(&ctrl.empty_q[i]), nact);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (!OUTPASS) asm volatile("griddepcontrol.wait;" ::: "memory");
  __syncthreads();

  if (warp >= C::NCW) {
    // ---------------- producer warp: lane 0 streams K,V; lane 1 streams Q ----------------
    const bool is_kv = (lane == 0);
    const uint32_t full = smem_u32(is_kv ? ctrl.full_kv : ctrl.full_q);
    const uint32_t empty = smem_u32(is_kv ? ctrl.empty_kv : ctrl.empty_q);
    const uint32_t base = is_kv ? kv_base : q_base;
    const int slot_bytes = is_kv ? C::KV_STAGE : C::T_STAGE;
    int S0 = R0;
    auto issue = [&](int st) {
      const int slot = st % C::NSTG;
      const uint32_t bar = full + 8u * slot;
      const uint32_t dst = base + slot * slot_bytes;
      const int y = S0 + st * C::SR;
      mbar_expect_tx(bar, (uint32_t)slot_bytes);
#pragma unroll
      for (int b = 0; b < C::NBOX; ++b) {
        const int x = h0 * D + 64 * b;
        if (is_kv) {
          tma_load_2d(dst + b * C::BOX_BYTES, &tmK, bar, x, y);
          tma_load_2d(dst + C::T_STAGE + b * C::BOX_BYTES, &tmV, bar, x, y);
        } else {
          tma_load_2d(dst + b * C::BOX_BYTES, &tmQ, bar, x, y);
        }
      }
    };
    __syncthreads();                                           // setup published (stream bounds)
    if (lane < 2) {
      S0 = ctrl.stream_begin;
      const int total = (OUTPASS && is_kv) ? 0 : (ctrl.stream_end - S0 + C::SR - 1) / C::SR;
      for (int st = 0; st < total; ++st) {
        if (st >= C::NSTG) mbar_wait(empty + 8u * (st % C::NSTG), (uint32_t)(((st / C::NSTG) - 1) & 1));
        issue(st);
      }
      for (int st = max(0, total - C::NSTG); st < total; ++st)      // no TMA may be in flight at exit
        mbar_wait(full + 8u * (st % C::NSTG), (uint32_t)((st / C::NSTG) & 1));
    }
    return;
  }

  // ---------------- consumer warps ----------------
  // A span table built once per scene (sla_build_span_table: SURVEY a1's work list) replaces the window search: one
  // 16-byte load instead of three dependent rounds of probes.  A table of another problem or launch geometry is ignored.
  bool planned = false;
  if (!OUTPASS && table != nullptr) {
    const int4 hdr = __ldg(table);
    planned = hdr.x == kSpanTableMagic && hdr.y == span && hdr.z == (int)gridDim.x && hdr.w == N;
  }
  if (planned) {
    if (threadIdx.x == 0) {
      const int4 rec = __ldg(table + 1 + sidx);              // (window of R0, stream begin, raw stream end, -)
      ctrl.wa = rec.x;
      ctrl.stream_begin = rec.y;
      ctrl.stream_end = max(rec.z, rec.y);
    }
  } else if (warp == 0) {
    int wa, wl;
    warp_windows_of_rows(off, W, R0, R1 - 1, wa, wl);
    if (lane == 0) {
      const int sa = __ldg(off + wa), ea = __ldg(off + wa + 1);
      const int sl = __ldg(off + wl), el = __ldg(off + wl + 1);
      // Ownership of a fused window (<= kFuseMax rows): the CTA whose span holds its MIDDLE row
      // (rows owned = span +- half a window at each end instead of a whole one: better balance).
      const int ma = sa + ((ea - sa) >> 1), ml = sl + ((el - sl) >> 1);
      int sb = (ea - sa <= kFuseMax) ? (ma >= R0 ? sa : ea) : R0;
      int se;
      if (el - sl <= kFuseMax) se = (ml < R1) ? el : sl;    // last window fused: owned iff its middle is here
      else se = R1;                                         // split: this CTA's piece ends at R1
      if (OUTPASS) {
        // span <= kFuseMax, so a split window that meets [R0,R1) holds R0 (window wa) or R1-1 (wl)
        const bool A = ea - sa > kFuseMax, B = el - sl > kFuseMax;
        sb = A ? R0 : (B ? max(sl, R0) : R0);
        se = B ? R1 : (A ? min(ea, R1) : sb);
      }
      ctrl.wa = wa;
      ctrl.stream_begin = sb;
      ctrl.stream_end = max(se, sb);
    }
  }
  __syncthreads();
  if (warp >= nact) return;

  const int hl = warp * C::HPW;                              // first head (within the slab) of this warp
  const int nh = min(C::HPW, nheads - hl);
  const int S0 = ctrl.stream_begin;
  const int total = (ctrl.stream_end - S0 + C::SR - 1) / C::SR;
  RingView kv = make_ring(kv_base, smem_u32(ctrl.full_kv), smem_u32(ctrl.empty_kv), C::NSTG);
  RingView qv = make_ring(q_base, smem_u32(ctrl.full_q), smem_u32(ctrl.empty_q), C::NSTG);
  T* out_head = out + (size_t)(h0 + hl) * D;

  // window walk with a 32-entry register cache of the offsets (one global round trip per 31 windows)
  int wbase = ctrl.wa;
  int cur = __ldg(off + min(wbase + lane, W));
  int nxt = __ldg(off + min(wbase + 31 + lane, W));
  auto bounds = [&](int w, int& s, int& e) {      // off[w], off[w+1]; w is non-decreasing across calls
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
  int w = wbase;
  if (OUTPASS) {
    while (w < W) {
      int s, e;
      bounds(w, s, e);
      if (s >= R1) break;
      if (e - s > kFuseMax) {
#pragma unroll
        for (int j = 0; j < C::HPW; ++j)
          if (j < nh) {
            const float* slot = ws + kWsHeaderFloats +
                                ((size_t)(s / (kFuseMax + 1)) * H + (h0 + hl + j)) * (size_t)((D + 1) * D);
            output_piece<D, MODE, T>(qv, hl + j, S0, max(s, R0), min(e, R1), e - s, slot, out_head + j * D, Ctot, eps);
          }
      }
      ++w;
    }
    ring_release_below<C::SR>(qv, total * C::SR);
  } else {
  while (w < W) {
    int s, e;
    bounds(w, s, e);
    if (s >= R1) break;
    const int m = e - s;
    if (m <= kFuseMax && s + (m >> 1) >= R1) break;               // middle beyond the span: a later CTA's
    if (m <= 0 || (m <= kFuseMax && s + (m >> 1) < R0)) { ++w; continue; }   // empty, or an earlier CTA's
    if (m <= QUAD_MAX) {
      // Pack the following whole short windows (owned, together <= 16 rows) into one 16-row tile.
      // Done for all cached windows at once: lane j holds off[wbase+j]; one ballot finds how many
      // consecutive windows fit, one OR-reduction builds the bit mask of window starts inside the
      // tile, and the window ordinal of tile row r is a popcount of that mask.
      const int i0 = w - wbase;                                   // lane of the first window (<= 30)
      const int e_j = __shfl_down_sync(0xffffffffu, cur, 1);      // off[wbase+lane+1]
      const int mid_j = cur + ((e_j - cur) >> 1);
      const bool fits = lane >= i0 && lane < 31 && (e_j - s) <= 16 && mid_j < R1;
      const unsigned okm = __ballot_sync(0xffffffffu, fits) >> i0;
      const int cnt = __ffs(~okm) - 1;                            // consecutive windows that fit (>= 1)
      const int rows = __shfl_sync(0xffffffffu, cur, i0 + cnt) - s;
      const unsigned startbit = (lane > i0 && lane < i0 + cnt) ? (1u << (cur - s)) : 0u;
      const unsigned starts = __reduce_or_sync(0xffffffffu, startbit) & 0xFFFEu;   // bit r: a window starts at row r
      const int wid = (lane < rows) ? __popc(starts & ((2u << lane) - 1u)) : -1;
      w += cnt;
      const int rel = s - S0;
      ring_release_below<C::SR>(kv, rel);
      ring_release_below<C::SR>(qv, rel);
      ring_wait_upto(kv, (rel + rows - 1) / C::SR);
      ring_wait_upto(qv, (rel + rows - 1) / C::SR);
#pragma unroll
      for (int j = 0; j < C::HPW; ++j)
        if (j < nh) quad_tile<D, MODE, T>(kv, qv, hl + j, rel, rows, wid, out_head + j * D + (size_t)s * Ctot, Ctot, eps);
      ring_release_below<C::SR>(kv, rel + rows);
      ring_release_below<C::SR>(qv, rel + rows);
      continue;
    }
    if (m <= kFuseMax) {
      process_window<D, MODE, false, T>(kv, qv, hl, nh, S0, s, e, out_head, Ctot, eps);
    } else if (ws != nullptr) {   // bounded entry (no workspace): a window that breaks the caller's promise is skipped
      float* slot = ws + kWsHeaderFloats + ((size_t)(s / (kFuseMax + 1)) * H + (h0 + hl)) * (size_t)((D + 1) * D);
      if (hl == 0 && lane == 0) reinterpret_cast<volatile int*>(ws)[0] = 1;   // tell the output kernel
      process_piece<D, MODE>(kv, hl, nh, S0, max(s, R0), min(e, R1), slot);
    }
    ++w;
  }
  // hand back every remaining stage the producers will issue (rows of split windows' Q, tail rows)
  ring_release_below<C::SR>(kv, total * C::SR);
  ring_release_below<C::SR>(qv, total * C::SR);
  }
}

// ---- span table ("chunk -> window map / work list", Fig. 3a) ----------------------------------
// One thread per window w = [s, e): the spans whose first row lies in the window get (w, stream begin), the spans whose
// last row lies in it get the stream end -- the very rules of the in-kernel search above, evaluated once per scene.
__global__ void __launch_bounds__(256)
sla_span_table_kernel(const int32_t* __restrict__ off, int N, int W, int span, int nx, int4* __restrict__ table) {
  asm volatile("griddepcontrol.launch_dependents;");
  asm volatile("griddepcontrol.wait;" ::: "memory");
  const int w = blockIdx.x * blockDim.x + threadIdx.x;
  if (w == 0) table[0] = make_int4(kSpanTableMagic, span, nx, N);
  if (w >= W) return;
  const int s = __ldg(off + w), e = __ldg(off + w + 1);
  if (e <= s) return;                                       // an empty window holds no row
  const int m = e - s, mid = s + (m >> 1);
  int* t = reinterpret_cast<int*>(table + 1);
  for (int sp = (s + span - 1) / span; sp < nx && sp * span < e; ++sp) {       // spans with R0 in [s, e)
    const int R0 = sp * span;
    t[4 * sp + 0] = w;
    t[4 * sp + 1] = (m <= kFuseMax) ? (mid >= R0 ? s : e) : R0;
  }
  for (int sp = s / span; sp < nx; ++sp) {                                      // spans with R1 - 1 in [s, e)
    const int R1 = min(sp * span + span, N);
    if (R1 - 1 < s) continue;
    if (R1 - 1 >= e) break;
    t[4 * sp + 2] = (m <= kFuseMax) ? (mid < R1 ? e : s) : R1;
    t[4 * sp + 3] = 0;
  }
}

// launch geometry of the main pass: rows per span and number of spans (shared by the kernel launch and the table)
template <int D>
void forward_geometry(int N, int H, int& span, int& nx) {
  const int slabs = (H + NW - 1) / NW;
  const int per_sm = (D == 16 ? 3 : 2);                     // resident CTAs per SM the grid is sized for
  nx = (per_sm * sm_count() + slabs - 1) / slabs;
  span = (N + nx - 1) / nx;
  if (span > 64) span = 64;             // short spans, several waves: dynamic balance across SMs
  span = (span + 15) / 16 * 16;
  if (span < 32) span = 32;
  nx = (N + span - 1) / span;
}

// ---- host side (tensor-map encoder, SM count: sla_tc_common.cuh) -----------------------------------
// `main_pass` = false: only the OUTPASS launch (the main pass was done by the tcgen05 kernel, sla_fwd_umma.cu,
// which follows the same workspace protocol).
template <int D, int MODE, typename T>
cudaError_t tc_launch(const Problem& p, cudaStream_t st, bool main_pass) {
  using C = Cfg<D>;
  CUtensorMap tq, tk, tv;
  const int Ctot = p.H * D;
  if (!make_map(&tq, p.q, p.N, Ctot, C::SR) || !make_map(&tk, p.k, p.N, Ctot, C::SR) ||
      !make_map(&tv, p.v, p.N, Ctot, C::SR))
    return cudaErrorInvalidValue;
  auto kern = sla_fwd_tc_kernel<D, MODE, T, false>;
  auto kern_out = sla_fwd_tc_kernel<D, MODE, T, true>;
  // the dynamic shared-memory opt-in is per device: set it once for every device this process uses
  static std::atomic<bool> attr_set[kMaxDevices];
  const int dev = current_device();
  if (!attr_set[dev].load(std::memory_order_acquire)) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_DYN);
    if (e == cudaSuccess)
      e = cudaFuncSetAttribute(kern_out, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_DYN);
    if (e != cudaSuccess) return e;
    attr_set[dev].store(true, std::memory_order_release);
  }
  const int slabs = (p.H + NW - 1) / NW;
  int span, nx;
  forward_geometry<D>(p.N, p.H, span, nx);
  dim3 grid(nx, slabs);
  // programmatic stream serialisation: see the note at the top of the kernel
  cudaLaunchAttribute pdl[1];
  pdl[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  pdl[0].val.programmaticStreamSerializationAllowed = 1;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid;
  cfg.blockDim = dim3(C::THREADS);
  cfg.dynamicSmemBytes = C::SMEM_DYN;
  cfg.stream = st;
  cfg.attrs = pdl;
  cfg.numAttrs = 1;
  if (main_pass) {
    cudaError_t le = cudaLaunchKernelEx(&cfg, kern, tq, tk, tv, p.off, (T*)p.out, p.ws_state, p.N, p.W, p.H, span, p.eps,
                                        (const int4*)p.span_table);
    if (le != cudaSuccess) return le;
  }
  if (!p.bounded) {
    // second pass: outputs of windows longer than kFuseMax (exits at once if there were none)
    const int span2 = kFuseMax / 16 * 16;   // the largest span OUTPASS handles: fewer CTAs to start and retire when nothing was split
    dim3 grid2((p.N + span2 - 1) / span2, slabs);
    cfg.gridDim = grid2;   // same attribute: resident behind the main kernel's tail, waits for its states
    cudaError_t le = cudaLaunchKernelEx(&cfg, kern_out, tq, tk, tv, p.off, (T*)p.out, p.ws_state, p.N, p.W, p.H,
                                        span2, p.eps, (const int4*)nullptr);
    if (le != cudaSuccess) return le;
  }
  return cudaGetLastError();
}

}  // namespace

bool forward_tc_supported(const Problem& p, int dt) {
  if (dt != SLA_F16 && dt != SLA_BF16) return false;
  if ((p.H * p.d) % 64 != 0) return false;                     // slab rows are whole 128-byte boxes
  return encode_fn() != nullptr;
}

size_t span_table_bytes(long long N, int H, int d) {
  int span, nx;
  if (d == 16) forward_geometry<16>((int)N, H, span, nx); else forward_geometry<32>((int)N, H, span, nx);
  return (size_t)(nx + 1) * sizeof(int4);
}

cudaError_t launch_span_table(const int32_t* off, int N, int W, int H, int d, void* table, cudaStream_t st) {
  int span, nx;
  if (d == 16) forward_geometry<16>(N, H, span, nx); else forward_geometry<32>(N, H, span, nx);
  cudaLaunchAttribute pdl[1];
  pdl[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  pdl[0].val.programmaticStreamSerializationAllowed = 1;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)((W + 255) / 256 > 0 ? (W + 255) / 256 : 1));
  cfg.blockDim = dim3(256);
  cfg.stream = st;
  cfg.attrs = pdl;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, sla_span_table_kernel, off, N, W, span, nx, (int4*)table);
}

cudaError_t launch_forward_tc(const Problem& p, int dt, cudaStream_t st) {
  bool main_pass = true;
  if (p.tcgen05) {   // main pass on tcgen05 (sla_fwd_umma.cu, same workspace protocol); long windows' outputs below
    cudaError_t e = launch_forward_umma_main(p, dt, st);
    if (e != cudaSuccess) return e;
    if (p.bounded) return cudaSuccess;
    main_pass = false;
  }
  // MODE = (bf16 ? 1 : 0) | (feature map << 1)
  const bool relu = p.phi == SLA_PHI_RELU;
  if (p.d == 16) {
    if (dt == SLA_F16) return relu ? tc_launch<16, 2, __half>(p, st, main_pass) : tc_launch<16, 0, __half>(p, st, main_pass);
    return relu ? tc_launch<16, 3, __nv_bfloat16>(p, st, main_pass) : tc_launch<16, 1, __nv_bfloat16>(p, st, main_pass);
  }
  if (dt == SLA_F16) return relu ? tc_launch<32, 2, __half>(p, st, main_pass) : tc_launch<32, 0, __half>(p, st, main_pass);
  return relu ? tc_launch<32, 3, __nv_bfloat16>(p, st, main_pass) : tc_launch<32, 1, __nv_bfloat16>(p, st, main_pass);
}

}  // namespace sla
