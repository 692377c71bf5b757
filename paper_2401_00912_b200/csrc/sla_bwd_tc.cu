// sla_bwd_tc.cu -- SLA backward for fp16 / bf16 I/O, d_h = 16, on sm_100a: same skeleton as the
// forward (sla_fwd_tc.cu): equal row spans per CTA, TMA + mbarrier rings, one consumer warp per head,
// mma.sync m16n8k16 with fp32 accumulation, window state in registers.
//
// Gradients of Eq. 3 (the paper is silent on backward), per window
// and head, a = phi(q), b = phi(k), g = dO:
//   pass A (K,V):    S = sum_j b_j^T v_j (kept as S^T fragments; operands that need S are block transposes), z = sum_j b_j
//   pass B (Q,dO):   num = a S, den = a.z, o = num/den, dnum = g/den, dden = -(g.o)/den
//                    dq = (dnum S^T + dden z) * phi'(q)
//                    dS += a^T dnum (kept as dS and dS^T fragments), dz += dden a
//   pass C (K,V):    dv = b dS,  dk = (v dS^T + dz) * phi'(k)
// Three streams (K,V / Q,dO / K,V again) run through three shared-memory rings.
//
// Scaling: with m rows and s = 2^-ceil(log2 m), the operands use S' = s S, z' = s z, so den' = s den
// and dnum' = g/den' = dnum/s stay O(1) in fp16; dS' = dS/s and dz' = dz/s are scaled back by s when
// they become operands of pass C.  Windows of <= 32 rows use split fp16 operands (hi + lo).
// Windows longer than kFuseMax rows are left to the three split passes at the end of this file (a flag in the
// workspace header tells them whether there is anything to do).
#include <cuda.h>

#include <atomic>

#include "sla_internal.cuh"

namespace sla {
namespace {

constexpr int NW = 8;     // consumer warps = heads per slab
constexpr int NST = 2;    // ring stages per stream
constexpr int BWD_PRECISE_MAX = 32;

template <int D> struct Cfg {
  static constexpr int SR = 32;                           // rows per ring stage
  static constexpr int NBOX = NW * D / 64;                // 128-byte column boxes per slab row
  static constexpr int BOX_BYTES = SR * 128;
  static constexpr int T_STAGE = NBOX * BOX_BYTES;        // one tensor's stage (8 KB at d_h = 16)
  static constexpr int KV_STAGE = 2 * T_STAGE;            // every ring stage holds two tensors
  static constexpr int RING_BYTES = 3 * NST * KV_STAGE;   // K,V | Q,dO | K,V again
  static constexpr int SMEM_DYN = RING_BYTES + 1024;
  static constexpr int THREADS = (NW + 1) * 32;
};

#include "sla_tc_common.cuh"

constexpr int D = 16;
using C = Cfg<D>;

// fragments of one (window, head); c index: rows g (c<2) / g+8 (c>=2), columns 2t + (c&1)
struct BwdState {
  float ST[2][4];    // S^T : rows r, column tile nt over p
  float Z[2][4];     // z[p] in columns p (same in every row)
  float dST[2][4];   // dS^T (scaled by 1/s)
  float DZ[2][4];    // dz   (scaled by 1/s)
  __device__ __forceinline__ void clear() {
#pragma unroll
    for (int a = 0; a < 2; ++a)
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        ST[a][c] = 0.f; Z[a][c] = 0.f; dST[a][c] = 0.f; DZ[a][c] = 0.f;
      }
  }
};

// B-operand pairs built from a 2-tile accumulator X[nt][c]:  op[n][b] = pack(X[b][2n], X[b][2n+1]) * scale
struct OpPair { uint32_t hi[2][2], lo[2][2]; };
template <bool PRECISE>
__device__ __forceinline__ void make_ops(const float (&X)[2][4], float scale, OpPair& o) {
#pragma unroll
  for (int n = 0; n < 2; ++n)
#pragma unroll
    for (int b = 0; b < 2; ++b) {
      const float x0 = X[b][2 * n] * scale, x1 = X[b][2 * n + 1] * scale;
      if (PRECISE) split_h2(x0, x1, o.hi[n][b], o.lo[n][b]);
      else { o.hi[n][b] = pack_h2(x0, x1); o.lo[n][b] = 0u; }
    }
}

// Operands of the transposed matrix: o holds the 8 x 8 blocks (output block n, contraction block b) of X; the same
// blocks of X^T are the movmatrix transposes of the blocks (b, n) of X.  Only S^T and dS^T are accumulated; the
// operands that need S and dS come from here.
__device__ __forceinline__ uint32_t movm_t(uint32_t x) {   // transpose of one 8x8 block of 16-bit elements
  uint32_t y;
  asm volatile("movmatrix.sync.aligned.m8n8.trans.b16 %0, %1;" : "=r"(y) : "r"(x));
  return y;
}
template <bool PRECISE>
__device__ __forceinline__ void transpose_ops(const OpPair& o, OpPair& t) {
#pragma unroll
  for (int n = 0; n < 2; ++n)
#pragma unroll
    for (int b = 0; b < 2; ++b) {
      t.hi[n][b] = movm_t(o.hi[b][n]);
      t.lo[n][b] = PRECISE ? movm_t(o.lo[b][n]) : 0u;
    }
}

// phi of a packed pair in fp32 (a) and its derivative factor: elu+1: (x>0 ? 1 : phi(x)); ReLU: [x > 0]
template <int MODE>
__device__ __forceinline__ void phi_pair(uint32_t raw, float2& a, float2& da) {
  constexpr bool BF16 = (MODE & 1) != 0;   // I/O dtype bf16
  constexpr int PHI = MODE >> 1;            // feature map (sla_feature_map_t)
  (void)BF16; (void)PHI;
  const float2 x = unpack2<BF16>(raw);
  if (PHI) {   // max(x, 0): phi' = [x > 0]
    da.x = x.x > 0.f ? 1.f : 0.f; da.y = x.y > 0.f ? 1.f : 0.f;
    a.x = fmaxf(x.x, 0.f); a.y = fmaxf(x.y, 0.f);
  } else {
    da.x = dphi_fast(x.x); da.y = dphi_fast(x.y);
    a.x = fmaxf(x.x, 0.f) + da.x; a.y = fmaxf(x.y, 0.f) + da.y;
  }
}
template <bool PRECISE>
__device__ __forceinline__ void to_op(float x0, float x1, uint32_t& hi, uint32_t& lo) {
  if (PRECISE) split_h2(x0, x1, hi, lo);
  else { hi = pack_h2(x0, x1); lo = 0u; }
}
// a (hi,lo) x b (hi,lo): 1 term, or the 3 leading terms
template <bool PRECISE>
__device__ __forceinline__ void mma3(float (&c)[4], const uint32_t (&ah)[4], const uint32_t (&al)[4],
                                     uint32_t bh0, uint32_t bh1, uint32_t bl0, uint32_t bl1) {
  mma16816(c, ah[0], ah[1], ah[2], ah[3], bh0, bh1);
  if (PRECISE) {
    mma16816(c, al[0], al[1], al[2], al[3], bh0, bh1);
    mma16816(c, ah[0], ah[1], ah[2], ah[3], bl0, bl1);
  }
}

// ReLU map only: with max(x, 0) a row's denominator can be eps alone, and g/den, dden reach 1/eps.  Every product that
// survives in the result then meets a zero factor (phi or phi' vanishes wherever the row's a.b did), so such
// intermediates only have to stay finite as fp16 operands: clamp them instead of letting them overflow to inf (0 * inf).
template <int PHI>
__device__ __forceinline__ float sat_h(float x) { return PHI ? fminf(fmaxf(x, -60000.f), 60000.f) : x; }

// ReLU map only: power-of-two rescaling of a tile's large intermediates.  `mx` = this lane's largest magnitude; returns k
// such that the warp-wide maximum times 2^-k is below 2^15 (k = 0 for the elu+1 map and for ordinary tiles), at most
// 10 so that the partner operand, phi(q) * 2^k, stays inside fp16.  The operand that carries 1/den is multiplied by
// 2^-k and its partner (or the fresh accumulator) by 2^k: exact.  What is still above fp16 after that belongs to rows
// whose denominator is eps alone (sat_h above).
template <int PHI>
__device__ __forceinline__ int tile_shift(float mx) {
  if (!PHI) return 0;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
  return min(10, max(0, (int)((__float_as_uint(mx) >> 23) & 0xffu) - 127 - 14));
}
__device__ __forceinline__ float pow2f(int k) { return __uint_as_float((uint32_t)(127 + k) << 23); }

// lane -> (tile row, 16-byte chunk select) for the x4 ldmatrix pattern
//   registers: (rows0-7,c0), (rows0-7,c1), (rows8-15,c0), (rows8-15,c1)
__device__ __forceinline__ void lane_pattern(int nvalid, int& trow, int& csel) {
  const int lane = threadIdx.x & 31, mi = lane >> 3;
  trow = (lane & 7) + 8 * (mi >> 1);
  if (trow >= nvalid) trow = 0;          // clamp: row 0 of the tile is always valid and loaded
  csel = mi & 1;
}

// ---- pass A: one 16-row K/V tile -> S^T, S, z -------------------------------------------------------
template <int MODE, bool PRECISE>
__device__ __forceinline__ void bwd_kv_tile(const RingView& rv, int hl, int rel0, int nvalid, BwdState& s) {
  constexpr bool BF16 = (MODE & 1) != 0;   // I/O dtype bf16
  constexpr int PHI = MODE >> 1;            // feature map (sla_feature_map_t)
  (void)BF16; (void)PHI;
  const int t = threadIdx.x & 3;
  int trow, csel;
  lane_pattern(nvalid, trow, csel);
  const int chunk = hl * 2 + csel;
  uint32_t kr[4], vr[4];
  ldsm_x4_t(ring_addr<D>(rv, C::KV_STAGE, 0, rel0 + trow, chunk), kr);
  ldsm_x4_t(ring_addr<D>(rv, C::KV_STAGE, C::T_STAGE, rel0 + trow, chunk), vr);
  // transposed loads: kr[i] = K[j = 2t,2t+1 (+8 for i>=2)][p = g (+8 for odd i)], same for vr with r
  uint32_t bh[4], bl[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int j0 = 2 * t + 8 * (i >> 1);
    if (PRECISE) {
      const float2 x = unpack2<BF16>(kr[i]);
      const float b0 = (j0 < nvalid) ? phi_fast<PHI>(x.x) : 0.f;
      const float b1 = (j0 + 1 < nvalid) ? phi_fast<PHI>(x.y) : 0.f;
      to_op<true>(b0, b1, bh[i], bl[i]);
    } else {   // long window: phi in fp16x2 (the operand is a single fp16 anyway), rows beyond the window zeroed
      bh[i] = phi_h2<BF16, PHI>(kr[i]);
      if (nvalid < 16) bh[i] &= pair_mask(j0, nvalid);
      bl[i] = 0u;
    }
  }
  if (BF16) {
#pragma unroll
    for (int i = 0; i < 4; ++i) { const float2 x = unpack2<true>(vr[i]); vr[i] = pack_h2(x.x, x.y); }
  }
  const uint32_t ones = 0x3C003C00u;
#pragma unroll
  for (int nt = 0; nt < 2; ++nt) {
    // S^T (rows r, cols p): A = V^T = (vr0..3), B = phi(K) tile nt = (b[nt], b[2+nt])
    mma16816(s.ST[nt], vr[0], vr[1], vr[2], vr[3], bh[nt], bh[2 + nt]);
    mma16816(s.Z[nt], ones, ones, ones, ones, bh[nt], bh[2 + nt]);
    if (PRECISE) {
      mma16816(s.ST[nt], vr[0], vr[1], vr[2], vr[3], bl[nt], bl[2 + nt]);
      mma16816(s.Z[nt], ones, ones, ones, ones, bl[nt], bl[2 + nt]);
    }
  }
}

struct PassBOps {
  OpPair num;            // from S^T: B operand of num = a S
  OpPair da;             // from S  : B operand of da = dnum S^T
  uint32_t zh[2], zl[2]; // z as B operand of den
  float zs[2][2];        // scaled z in columns p = 8*np + 2t + c
  float eps;             // epsilon of the denominator on the scale of the operands (eps * s); 0 for elu+1
};

// ---- pass B: one 16-row Q/dO tile -> dq rows, dS^T, dS, dz accumulators ------------------------------
template <int MODE, bool PRECISE, typename T>
__device__ __forceinline__ void bwd_q_tile(const RingView& rv, int hl, int rel0, int nvalid,
                                           const PassBOps& op, BwdState& s, T* __restrict__ dq_rows,
                                           int C_total) {
  constexpr bool BF16 = (MODE & 1) != 0;   // I/O dtype bf16
  constexpr int PHI = MODE >> 1;            // feature map (sla_feature_map_t)
  (void)BF16; (void)PHI;
  const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
  int trow, csel;
  lane_pattern(nvalid, trow, csel);
  const int chunk = hl * 2 + csel;
  const int perm[4] = {0, 2, 1, 3};   // ldmatrix register order -> A-fragment order (a0..a3)
  uint32_t qn[4], gn[4];
  ldsm_x4(ring_addr<D>(rv, C::KV_STAGE, 0, rel0 + trow, chunk), qn);
  ldsm_x4(ring_addr<D>(rv, C::KV_STAGE, C::T_STAGE, rel0 + trow, chunk), gn);
  // A fragments: index 0: (row g, cols 2t..), 1: (row g+8, cols 2t..), 2: (row g, cols 8+2t..), 3: (row g+8, 8+2t..)
  uint32_t ah[4], al[4], dph2[4];   // dph2: phi'(q) as fp16x2 (long windows)
  float2 dph[4], gv[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    if (PRECISE) {
      float2 a;
      phi_pair<MODE>(qn[perm[i]], a, dph[i]);
      to_op<true>(a.x, a.y, ah[i], al[i]);
    } else {
      phi_dphi_h2<BF16, PHI>(qn[perm[i]], ah[i], dph2[i]);
      al[i] = 0u;
    }
    gv[i] = unpack2<BF16>(gn[perm[i]]);
  }
  float num[2][4] = {{0.f, 0.f, 0.f, 0.f}, {0.f, 0.f, 0.f, 0.f}}, den[4] = {0.f, 0.f, 0.f, 0.f};
  mma3<PRECISE>(den, ah, al, op.zh[0], op.zh[1], op.zl[0], op.zl[1]);
#pragma unroll
  for (int n = 0; n < 2; ++n) mma3<PRECISE>(num[n], ah, al, op.num.hi[n][0], op.num.hi[n][1], op.num.lo[n][0], op.num.lo[n][1]);
  const float inv0 = fast_rcp(PHI ? den[0] + op.eps : den[0]), inv1 = fast_rcp(PHI ? den[2] + op.eps : den[2]);   // rows g, g+8
  // g.o per row: this lane holds columns 2t,2t+1 (tile 0) and 8+2t.. (tile 1) of rows g and g+8
  float go0 = gv[0].x * num[0][0] + gv[0].y * num[0][1] + gv[2].x * num[1][0] + gv[2].y * num[1][1];
  float go1 = gv[1].x * num[0][2] + gv[1].y * num[0][3] + gv[3].x * num[1][2] + gv[3].y * num[1][3];
  go0 += __shfl_xor_sync(0xffffffffu, go0, 1); go0 += __shfl_xor_sync(0xffffffffu, go0, 2);
  go1 += __shfl_xor_sync(0xffffffffu, go1, 1); go1 += __shfl_xor_sync(0xffffffffu, go1, 2);
  const float dden0 = -(go0 * inv0) * inv0, dden1 = -(go1 * inv1) * inv1;   // o = num*inv
  // ReLU: rows whose denominator is almost eps alone make g/den and dden huge; rescale the tile by a power of two
  float gmax = 0.f;
  if (PHI) {
#pragma unroll
    for (int i = 0; i < 4; ++i) gmax = fmaxf(gmax, fmaxf(fabsf(gv[i].x), fabsf(gv[i].y)) * ((i & 1) ? inv1 : inv0));
    gmax = fmaxf(gmax, fmaxf(fabsf(dden0), fabsf(dden1)));
  }
  const int ksh = tile_shift<PHI>(gmax);
  const float dn = pow2f(-ksh), up = pow2f(ksh);        // both 1 unless ReLU and an ill-conditioned row
  // dnum as A fragment (rows g / g+8 scaled by their 1/den)
  uint32_t dh[4], dl[4];
  if (PRECISE || BF16 || PHI) {
    const float i0 = PHI ? inv0 * dn : inv0, i1 = PHI ? inv1 * dn : inv1;
    to_op<PRECISE>(sat_h<PHI>(gv[0].x * i0), sat_h<PHI>(gv[0].y * i0), dh[0], dl[0]);
    to_op<PRECISE>(sat_h<PHI>(gv[1].x * i1), sat_h<PHI>(gv[1].y * i1), dh[1], dl[1]);
    to_op<PRECISE>(sat_h<PHI>(gv[2].x * i0), sat_h<PHI>(gv[2].y * i0), dh[2], dl[2]);
    to_op<PRECISE>(sat_h<PHI>(gv[3].x * i1), sat_h<PHI>(gv[3].y * i1), dh[3], dl[3]);
  } else {   // fp16 dO, long window: scale the packed pairs directly
    const uint32_t i0h = pack_h2(inv0, inv0), i1h = pack_h2(inv1, inv1);
    dh[0] = hmul2_u32(gn[perm[0]], i0h); dh[1] = hmul2_u32(gn[perm[1]], i1h);
    dh[2] = hmul2_u32(gn[perm[2]], i0h); dh[3] = hmul2_u32(gn[perm[3]], i1h);
    dl[0] = dl[1] = dl[2] = dl[3] = 0u;
  }
  // da = dnum S^T + dden z ; dq = da * phi'(q)
#pragma unroll
  for (int np = 0; np < 2; ++np) {
    float da[4] = {0.f, 0.f, 0.f, 0.f};
    mma3<PRECISE>(da, dh, dl, op.da.hi[np][0], op.da.hi[np][1], op.da.lo[np][0], op.da.lo[np][1]);
    // C fragment (np): c0,c1 = (row g, p = 8np+2t,+1) <-> A index 2*np ; c2,c3 = row g+8 <-> A index 2*np+1
    if (PHI) { da[0] *= up; da[1] *= up; da[2] *= up; da[3] *= up; }
    const float q0 = da[0] + dden0 * op.zs[np][0], q1 = da[1] + dden0 * op.zs[np][1];
    const float q2 = da[2] + dden1 * op.zs[np][0], q3 = da[3] + dden1 * op.zs[np][1];
    uint32_t* p0 = reinterpret_cast<uint32_t*>(dq_rows + (size_t)g * C_total + 8 * np + 2 * t);
    uint32_t* p1 = reinterpret_cast<uint32_t*>(dq_rows + (size_t)(g + 8) * C_total + 8 * np + 2 * t);
    if (PRECISE) {
      if (g < nvalid) *p0 = pack_out<BF16>(q0 * dph[2 * np].x, q1 * dph[2 * np].y);
      if (g + 8 < nvalid) *p1 = pack_out<BF16>(q2 * dph[2 * np + 1].x, q3 * dph[2 * np + 1].y);
    } else {
      if (g < nvalid) *p0 = pack_out_times_h2<BF16, PHI != 0>(q0, q1, dph2[2 * np]);
      if (g + 8 < nvalid) *p1 = pack_out_times_h2<BF16, PHI != 0>(q2, q3, dph2[2 * np + 1]);
    }
  }
  // ---- transposed operands (contraction over the rows i of the tile) ----
  uint32_t qt[4], gt[4];
  ldsm_x4_t(ring_addr<D>(rv, C::KV_STAGE, 0, rel0 + trow, chunk), qt);
  ldsm_x4_t(ring_addr<D>(rv, C::KV_STAGE, C::T_STAGE, rel0 + trow, chunk), gt);
  // qt[i] = Q[i' = 2t,2t+1 (+8 for i>=2)][p = g (+8 for odd i)] ; gt[i] likewise with r
  // 1/den and dden of rows 2t, 2t+1, 2t+8, 2t+9 live in the lanes whose g equals that row
  const int l0 = 4 * (2 * t), l1 = 4 * (2 * t + 1);
  const float ir0 = __shfl_sync(0xffffffffu, inv0, l0), ir1 = __shfl_sync(0xffffffffu, inv0, l1);
  const float ir2 = __shfl_sync(0xffffffffu, inv1, l0), ir3 = __shfl_sync(0xffffffffu, inv1, l1);
  float dd0 = __shfl_sync(0xffffffffu, dden0, l0), dd1 = __shfl_sync(0xffffffffu, dden0, l1);
  float dd2 = __shfl_sync(0xffffffffu, dden1, l0), dd3 = __shfl_sync(0xffffffffu, dden1, l1);
  uint32_t uh[4], ul[4], th[4], tl[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int i0 = 2 * t + 8 * (i >> 1);
    const float s0 = ((i >> 1) ? ir2 : ir0) * dn, s1 = ((i >> 1) ? ir3 : ir1) * dn;   // dn = 1 unless ReLU
    if (PRECISE) {
      const float2 x = unpack2<BF16>(qt[i]);
      const float a0 = (i0 < nvalid) ? phi_fast<PHI>(x.x) : 0.f;       // rows beyond the window contribute nothing
      const float a1 = (i0 + 1 < nvalid) ? phi_fast<PHI>(x.y) : 0.f;
      to_op<true>(sat_h<PHI>(a0 * up), sat_h<PHI>(a1 * up), uh[i], ul[i]);
    } else {
      uh[i] = phi_h2<BF16, PHI>(qt[i]);
      if (nvalid < 16) uh[i] &= pair_mask(i0, nvalid);
      if (PHI) uh[i] = hmul2_u32(uh[i], pack_h2(up, up));
      ul[i] = 0u;
    }
    if (PRECISE || BF16 || PHI) {
      const float2 gg = unpack2<BF16>(gt[i]);
      to_op<PRECISE>(sat_h<PHI>(gg.x * s0), sat_h<PHI>(gg.y * s1), th[i], tl[i]);
    } else {
      th[i] = hmul2_u32(gt[i], pack_h2(s0, s1));
      tl[i] = 0u;
    }
  }
  uint32_t ddh[2], ddl[2];
  to_op<PRECISE>(sat_h<PHI>(dd0 * dn), sat_h<PHI>(dd1 * dn), ddh[0], ddl[0]);
  to_op<PRECISE>(sat_h<PHI>(dd2 * dn), sat_h<PHI>(dd3 * dn), ddh[1], ddl[1]);
  const uint32_t dda_h[4] = {ddh[0], ddh[0], ddh[1], ddh[1]}, dda_l[4] = {ddl[0], ddl[0], ddl[1], ddl[1]};
#pragma unroll
  for (int nt = 0; nt < 2; ++nt) {
    // dS^T (rows r, cols p): A = dnum^T = (t0..3), B = a tile nt over p = (u[nt], u[2+nt])
    mma3<PRECISE>(s.dST[nt], th, tl, uh[nt], uh[2 + nt], ul[nt], ul[2 + nt]);
    // dz[p] = sum_i dden_i a_i[p]: A rows all equal to dden over i, B = a tile nt
    mma3<PRECISE>(s.DZ[nt], dda_h, dda_l, uh[nt], uh[2 + nt], ul[nt], ul[2 + nt]);
  }
}

struct PassCOps {
  OpPair dv;             // from dS^T: B operand of dv = b dS
  OpPair db;             // from dS  : B operand of db = v dS^T
  float dzs[2][2];       // dz in columns p = 8*np + 2t + c
};

// ---- pass C: one 16-row K/V tile -> dk, dv rows ------------------------------------------------------
template <int MODE, bool PRECISE, typename T>
__device__ __forceinline__ void bwd_kv_out_tile(const RingView& rv, int hl, int rel0, int nvalid,
                                                const PassCOps& op, T* __restrict__ dk_rows,
                                                T* __restrict__ dv_rows, int C_total) {
  constexpr bool BF16 = (MODE & 1) != 0;   // I/O dtype bf16
  constexpr int PHI = MODE >> 1;            // feature map (sla_feature_map_t)
  (void)BF16; (void)PHI;
  const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
  int trow, csel;
  lane_pattern(nvalid, trow, csel);
  const int chunk = hl * 2 + csel;
  const int perm[4] = {0, 2, 1, 3};
  uint32_t kn[4], vn[4];
  ldsm_x4(ring_addr<D>(rv, C::KV_STAGE, 0, rel0 + trow, chunk), kn);
  ldsm_x4(ring_addr<D>(rv, C::KV_STAGE, C::T_STAGE, rel0 + trow, chunk), vn);
  uint32_t bh[4], bl[4], vh[4], dph2[4];
  float2 dph[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    if (PRECISE) {
      float2 b;
      phi_pair<MODE>(kn[perm[i]], b, dph[i]);
      to_op<true>(b.x, b.y, bh[i], bl[i]);
    } else {
      phi_dphi_h2<BF16, PHI>(kn[perm[i]], bh[i], dph2[i]);
      bl[i] = 0u;
    }
    if (BF16) { const float2 x = unpack2<true>(vn[perm[i]]); vh[i] = pack_h2(x.x, x.y); }
    else vh[i] = vn[perm[i]];
  }
#pragma unroll
  for (int n = 0; n < 2; ++n) {
    float dv[4] = {0.f, 0.f, 0.f, 0.f}, db[4] = {0.f, 0.f, 0.f, 0.f};
    mma3<PRECISE>(dv, bh, bl, op.dv.hi[n][0], op.dv.hi[n][1], op.dv.lo[n][0], op.dv.lo[n][1]);
    mma16816(db, vh[0], vh[1], vh[2], vh[3], op.db.hi[n][0], op.db.hi[n][1]);
    if (PRECISE) mma16816(db, vh[0], vh[1], vh[2], vh[3], op.db.lo[n][0], op.db.lo[n][1]);   // v is exact
    const float k0 = db[0] + op.dzs[n][0], k1 = db[1] + op.dzs[n][1];
    const float k2 = db[2] + op.dzs[n][0], k3 = db[3] + op.dzs[n][1];
    const size_t o0 = (size_t)g * C_total + 8 * n + 2 * t, o1 = (size_t)(g + 8) * C_total + 8 * n + 2 * t;
    if (g < nvalid) {
      *reinterpret_cast<uint32_t*>(dv_rows + o0) = pack_out<BF16>(dv[0], dv[1]);
      *reinterpret_cast<uint32_t*>(dk_rows + o0) = PRECISE ? pack_out<BF16>(k0 * dph[2 * n].x, k1 * dph[2 * n].y)
                                                           : pack_out_times_h2<BF16, PHI != 0>(k0, k1, dph2[2 * n]);
    }
    if (g + 8 < nvalid) {
      *reinterpret_cast<uint32_t*>(dv_rows + o1) = pack_out<BF16>(dv[2], dv[3]);
      *reinterpret_cast<uint32_t*>(dk_rows + o1) = PRECISE ? pack_out<BF16>(k2 * dph[2 * n + 1].x, k3 * dph[2 * n + 1].y)
                                                           : pack_out_times_h2<BF16, PHI != 0>(k2, k3, dph2[2 * n + 1]);
    }
  }
}

// ---- packed short windows: the backward of the masked quadratic form inside one 16-row tile ---------------------
// Several WHOLE windows of <= 16 rows each, together <= 16 consecutive rows (the forward's packing).  With
// P_ij = a_i.b_j masked to same-window pairs, r_i = sum_j P_ij, W = P / r, o_i = sum_j W_ij v_j (the
// same function as Eq. 3) and g = dO:
//   X_ij = g_i.v_j,   g_i.o_i = sum_j W_ij X_ij,   dP_ij = (X_ij - g_i.o_i) / r_i  (masked)
//   dv_j = sum_i W_ij g_i,   da_i = sum_j dP_ij b_j,   db_j = sum_i dP_ij a_i,   dq = da phi'(q),  dk = db phi'(k)
// a, b, W and dP are split into fp16 hi+lo operands (as in the forward's packed tiles); g and v are exact.
// `wid` = window ordinal of tile row `lane` (lanes >= nvalid hold -1).
template <int MODE, typename T>
__device__ __forceinline__ void bwd_quad_tile(const RingView& kv, const RingView& qg, int hl, int rel0, int nvalid,
                                              int wid, T* __restrict__ dq_rows, T* __restrict__ dk_rows,
                                              T* __restrict__ dv_rows, int C_total, float eps) {
  constexpr bool BF16 = (MODE & 1) != 0;   // I/O dtype bf16
  constexpr int PHI = MODE >> 1;            // feature map (sla_feature_map_t)
  (void)BF16; (void)PHI;
  const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
  int trow, csel;
  lane_pattern(nvalid, trow, csel);
  const int chunk = hl * 2 + csel;
  const int perm[4] = {0, 2, 1, 3};   // ldmatrix register order -> A-fragment order
  uint32_t rq[4], rk[4], rg[4], rv[4], tq[4], tk[4], tg[4];
  ldsm_x4(ring_addr<D>(qg, C::KV_STAGE, 0, rel0 + trow, chunk), rq);
  ldsm_x4(ring_addr<D>(qg, C::KV_STAGE, C::T_STAGE, rel0 + trow, chunk), rg);
  ldsm_x4(ring_addr<D>(kv, C::KV_STAGE, 0, rel0 + trow, chunk), rk);
  ldsm_x4(ring_addr<D>(kv, C::KV_STAGE, C::T_STAGE, rel0 + trow, chunk), rv);
  ldsm_x4_t(ring_addr<D>(qg, C::KV_STAGE, 0, rel0 + trow, chunk), tq);
  ldsm_x4_t(ring_addr<D>(qg, C::KV_STAGE, C::T_STAGE, rel0 + trow, chunk), tg);
  ldsm_x4_t(ring_addr<D>(kv, C::KV_STAGE, 0, rel0 + trow, chunk), tk);
  // operands: a (A of P), b (B of P), aT (B of db), bT (B of da); derivative factors in the ldmatrix block order
  uint32_t ah[4], al[4], bh[4], bl[4], ath[4], atl[4], bth[4], btl[4], gh[4], vh[4], gth[4];
  float2 dpq[4], dpk[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    float2 a, b, x, da_, db_;
    phi_pair<MODE>(rq[i], a, dpq[i]);
    phi_pair<MODE>(rk[i], b, dpk[i]);
    split_h2(a.x, a.y, ah[i], al[i]);
    split_h2(b.x, b.y, bh[i], bl[i]);
    phi_pair<MODE>(tq[i], x, da_);
    split_h2(x.x, x.y, ath[i], atl[i]);
    phi_pair<MODE>(tk[i], x, db_);
    split_h2(x.x, x.y, bth[i], btl[i]);
    if (BF16) {
      float2 y = unpack2<true>(rg[i]); gh[i] = pack_h2(y.x, y.y);
      y = unpack2<true>(rv[i]); vh[i] = pack_h2(y.x, y.y);
      y = unpack2<true>(tg[i]); gth[i] = pack_h2(y.x, y.y);
    } else { gh[i] = rg[i]; vh[i] = rv[i]; gth[i] = tg[i]; }
  }
  const uint32_t aH[4] = {ah[0], ah[2], ah[1], ah[3]}, aL[4] = {al[0], al[2], al[1], al[3]};
  const uint32_t gA[4] = {gh[perm[0]], gh[perm[1]], gh[perm[2]], gh[perm[3]]};
  // P[jt][c] and X[jt][c]: rows i = g (c<2) / g+8 (c>=2), columns j = 8 jt + 2t + (c&1)
  float P[2][4] = {{0.f, 0.f, 0.f, 0.f}, {0.f, 0.f, 0.f, 0.f}}, X[2][4] = {{0.f, 0.f, 0.f, 0.f}, {0.f, 0.f, 0.f, 0.f}};
#pragma unroll
  for (int jt = 0; jt < 2; ++jt) {
    mma3<true>(P[jt], aH, aL, bh[2 * jt], bh[2 * jt + 1], bl[2 * jt], bl[2 * jt + 1]);
    mma16816(X[jt], gA[0], gA[1], gA[2], gA[3], vh[2 * jt], vh[2 * jt + 1]);
  }
  const int wi0 = __shfl_sync(0xffffffffu, wid, g), wi1 = __shfl_sync(0xffffffffu, wid, g + 8);
  float rs0 = 0.f, rs1 = 0.f;
  unsigned same = 0u;                         // bit 2 jt + c: pair (row g, column j) in one window; bit 4 + ..: row g+8
#pragma unroll
  for (int jt = 0; jt < 2; ++jt)
#pragma unroll
    for (int c = 0; c < 2; ++c) {
      const int wj = __shfl_sync(0xffffffffu, wid, 8 * jt + 2 * t + c);
      const bool m0 = wj == wi0 && wj >= 0, m1 = wj == wi1 && wj >= 0;
      same |= (m0 ? 1u : 0u) << (2 * jt + c) | (m1 ? 1u : 0u) << (4 + 2 * jt + c);
      P[jt][c] = m0 ? P[jt][c] : 0.f;          X[jt][c] = m0 ? X[jt][c] : 0.f;
      P[jt][2 + c] = m1 ? P[jt][2 + c] : 0.f;  X[jt][2 + c] = m1 ? X[jt][2 + c] : 0.f;
      rs0 += P[jt][c];
      rs1 += P[jt][2 + c];
    }
  rs0 += __shfl_xor_sync(0xffffffffu, rs0, 1); rs0 += __shfl_xor_sync(0xffffffffu, rs0, 2);
  rs1 += __shfl_xor_sync(0xffffffffu, rs1, 1); rs1 += __shfl_xor_sync(0xffffffffu, rs1, 2);
  const float inv0 = (g < nvalid) ? fast_rcp(PHI ? rs0 + eps : rs0) : 0.f;
  const float inv1 = (g + 8 < nvalid) ? fast_rcp(PHI ? rs1 + eps : rs1) : 0.f;
  float go0 = 0.f, go1 = 0.f;                 // g_i . o_i = sum_j W_ij X_ij
#pragma unroll
  for (int jt = 0; jt < 2; ++jt)
#pragma unroll
    for (int c = 0; c < 2; ++c) {
      P[jt][c] *= inv0; P[jt][2 + c] *= inv1;             // W
      go0 += P[jt][c] * X[jt][c];
      go1 += P[jt][2 + c] * X[jt][2 + c];
    }
  go0 += __shfl_xor_sync(0xffffffffu, go0, 1); go0 += __shfl_xor_sync(0xffffffffu, go0, 2);
  go1 += __shfl_xor_sync(0xffffffffu, go1, 1); go1 += __shfl_xor_sync(0xffffffffu, go1, 2);
#pragma unroll
  for (int jt = 0; jt < 2; ++jt)
#pragma unroll
    for (int c = 0; c < 2; ++c) {               // dP, zero on masked pairs (a ReLU weight can be 0 on an unmasked one)
      X[jt][c] = ((same >> (2 * jt + c)) & 1u) ? (X[jt][c] - go0) * inv0 : 0.f;
      X[jt][2 + c] = ((same >> (4 + 2 * jt + c)) & 1u) ? (X[jt][2 + c] - go1) * inv1 : 0.f;
    }
  // ReLU: a row whose weights sum to almost eps alone has dP of the order 1/eps; rescale the tile by a power of two
  float pmax = 0.f;
  if (PHI) {
#pragma unroll
    for (int jt = 0; jt < 2; ++jt)
#pragma unroll
      for (int c = 0; c < 4; ++c) pmax = fmaxf(pmax, fabsf(X[jt][c]));
  }
  const int ksh = tile_shift<PHI>(pmax);
  const float up = pow2f(ksh);
  if (PHI) {
    const float dn = pow2f(-ksh);
#pragma unroll
    for (int jt = 0; jt < 2; ++jt)
#pragma unroll
      for (int c = 0; c < 4; ++c) X[jt][c] = sat_h<PHI>(X[jt][c] * dn);
  }
  // A operands (k = j) of W and dP, and their transposes (m = j, k = i) by 8x8 block transposes
  uint32_t wh[4], wl[4], ph[4], pl[4], wth[4], wtl[4], pth[4], ptl[4];
#pragma unroll
  for (int jt = 0; jt < 2; ++jt)
#pragma unroll
    for (int ib = 0; ib < 2; ++ib) {
      split_h2(P[jt][2 * ib], P[jt][2 * ib + 1], wh[2 * jt + ib], wl[2 * jt + ib]);   // A index: a0=(g,jt0) a1=(g+8,jt0) a2=(g,jt1) a3=(g+8,jt1)
      split_h2(X[jt][2 * ib], X[jt][2 * ib + 1], ph[2 * jt + ib], pl[2 * jt + ib]);
    }
  // block (ib, jt) sits at A index 2 jt + ib; its transpose is the block (jt, ib) of the transposed operand: index 2 ib + jt
#pragma unroll
  for (int jt = 0; jt < 2; ++jt)
#pragma unroll
    for (int ib = 0; ib < 2; ++ib) {
      wth[2 * ib + jt] = movm_t(wh[2 * jt + ib]); wtl[2 * ib + jt] = movm_t(wl[2 * jt + ib]);
      pth[2 * ib + jt] = movm_t(ph[2 * jt + ib]); ptl[2 * ib + jt] = movm_t(pl[2 * jt + ib]);
    }
#pragma unroll
  for (int nt = 0; nt < 2; ++nt) {
    // dv (rows j, cols r): A = W^T, B = g over rows i (transposed load): exact operand
    float dv[4] = {0.f, 0.f, 0.f, 0.f}, da[4] = {0.f, 0.f, 0.f, 0.f}, db[4] = {0.f, 0.f, 0.f, 0.f};
    mma16816(dv, wth[0], wth[1], wth[2], wth[3], gth[nt], gth[2 + nt]);
    mma16816(dv, wtl[0], wtl[1], wtl[2], wtl[3], gth[nt], gth[2 + nt]);
    // da (rows i, cols p): A = dP, B = b over rows j ; db (rows j, cols p): A = dP^T, B = a over rows i
    mma3<true>(da, ph, pl, bth[nt], bth[2 + nt], btl[nt], btl[2 + nt]);
    mma3<true>(db, pth, ptl, ath[nt], ath[2 + nt], atl[nt], atl[2 + nt]);
    if (PHI) {
#pragma unroll
      for (int c = 0; c < 4; ++c) { da[c] *= up; db[c] *= up; }
    }
    // derivative factors at (row g / g+8, channels 8 nt + 2t..): ldmatrix blocks (rowhalf, chalf = nt) = index 2*rowhalf + nt
    const size_t o0 = (size_t)g * C_total + 8 * nt + 2 * t, o1 = (size_t)(g + 8) * C_total + 8 * nt + 2 * t;
    if (g < nvalid) {
      *reinterpret_cast<uint32_t*>(dv_rows + o0) = pack_out<BF16>(dv[0], dv[1]);
      *reinterpret_cast<uint32_t*>(dq_rows + o0) = pack_out<BF16>(da[0] * dpq[nt].x, da[1] * dpq[nt].y);
      *reinterpret_cast<uint32_t*>(dk_rows + o0) = pack_out<BF16>(db[0] * dpk[nt].x, db[1] * dpk[nt].y);
    }
    if (g + 8 < nvalid) {
      *reinterpret_cast<uint32_t*>(dv_rows + o1) = pack_out<BF16>(dv[2], dv[3]);
      *reinterpret_cast<uint32_t*>(dq_rows + o1) = pack_out<BF16>(da[2] * dpq[2 + nt].x, da[3] * dpq[2 + nt].y);
      *reinterpret_cast<uint32_t*>(dk_rows + o1) = pack_out<BF16>(db[2] * dpk[2 + nt].x, db[3] * dpk[2 + nt].y);
    }
  }
}

// ---- one whole window: the three passes -------------------------------------------------------------
template <int MODE, bool PRECISE, typename T>
__device__ __forceinline__ void bwd_window(RingView& kv, RingView& qg, RingView& kv2, int hl, int S0, int s,
                                           int e, T* __restrict__ dq_head, T* __restrict__ dk_head,
                                           T* __restrict__ dv_head, int Ctot, float eps) {
  constexpr bool BF16 = (MODE & 1) != 0;   // I/O dtype bf16
  constexpr int PHI = MODE >> 1;            // feature map (sla_feature_map_t)
  (void)BF16; (void)PHI;
  BwdState st;
  st.clear();
  for (int r = s; r < e; r += 16) {
    const int nv = min(16, e - r), rel = r - S0;
    ring_release_below<C::SR>(kv, rel);
    ring_wait_upto(kv, (rel + nv - 1) / C::SR);
    bwd_kv_tile<MODE, PRECISE>(kv, hl, rel, nv, st);
  }
  const float scale = z_scale<2>(st.Z);                   // s: largest z of the window -> [1, 2) (sla_tc_base.cuh)
  PassBOps ob;
  ob.eps = eps * scale;
  make_ops<PRECISE>(st.ST, scale, ob.num);
  transpose_ops<PRECISE>(ob.num, ob.da);
#pragma unroll
  for (int b = 0; b < 2; ++b) {
    ob.zs[b][0] = st.Z[b][0] * scale; ob.zs[b][1] = st.Z[b][1] * scale;
    to_op<PRECISE>(ob.zs[b][0], ob.zs[b][1], ob.zh[b], ob.zl[b]);
  }
  for (int r = s; r < e; r += 16) {
    const int nv = min(16, e - r), rel = r - S0;
    ring_release_below<C::SR>(qg, rel);
    ring_wait_upto(qg, (rel + nv - 1) / C::SR);
    bwd_q_tile<MODE, PRECISE, T>(qg, hl, rel, nv, ob, st, dq_head + (size_t)r * Ctot, Ctot);
  }
  PassCOps oc;
  make_ops<PRECISE>(st.dST, scale, oc.dv);
  transpose_ops<PRECISE>(oc.dv, oc.db);
#pragma unroll
  for (int b = 0; b < 2; ++b) { oc.dzs[b][0] = st.DZ[b][0] * scale; oc.dzs[b][1] = st.DZ[b][1] * scale; }
  for (int r = s; r < e; r += 16) {
    const int nv = min(16, e - r), rel = r - S0;
    ring_release_below<C::SR>(kv2, rel);
    ring_wait_upto(kv2, (rel + nv - 1) / C::SR);
    bwd_kv_out_tile<MODE, PRECISE, T>(kv2, hl, rel, nv, oc, dk_head + (size_t)r * Ctot,
                                      dv_head + (size_t)r * Ctot, Ctot);
  }
}

struct Ctrl {
  unsigned long long full[3][NST], empty[3][NST];
  int wa, stream_begin, stream_end;
};

template <int MODE, typename T>
__global__ void __launch_bounds__(Cfg<D>::THREADS, 2)
sla_bwd_tc_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmK,
                  const __grid_constant__ CUtensorMap tmV, const __grid_constant__ CUtensorMap tmG,
                  const int32_t* __restrict__ off, T* __restrict__ dq, T* __restrict__ dk,
                  T* __restrict__ dv, float* __restrict__ ws, int N, int W, int H, int span, float eps) {
  constexpr bool BF16 = (MODE & 1) != 0;   // I/O dtype bf16
  constexpr int PHI = MODE >> 1;            // feature map (sla_feature_map_t)
  (void)BF16; (void)PHI;
  extern __shared__ uint8_t dyn_smem[];
  __shared__ Ctrl ctrl;
  // programmatic dependent launch, as the forward: resident behind the previous kernel's tail, barrier set-up runs
  // ahead, nothing that kernel may have written is touched before griddepcontrol.wait
  asm volatile("griddepcontrol.launch_dependents;");
  const uint32_t ring = (smem_u32(dyn_smem) + 1023u) & ~1023u;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int nspan = gridDim.x, bx = blockIdx.x;
  const int sidx = (bx & 1) ? nspan - 1 - (bx >> 1) : (bx >> 1);     // outside-in, as the forward
  const int R0 = sidx * span, R1 = min(R0 + span, N);
  const int h0 = blockIdx.y * NW;
  const int nheads = min(NW, H - h0);
  const int Ctot = H * D;

  if (threadIdx.x == 0) {
    for (int r = 0; r < 3; ++r)
      for (int i = 0; i < NST; ++i) {
        mbar_init(smem_u32(&ctrl.full[r][i]), 1);
        mbar_init(smem_u32(&ctrl.empty[r][i]), nheads);
      }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  asm volatile("griddepcontrol.wait;" ::: "memory");
  __syncthreads();

  if (warp >= NW) {
    // producer warp: lane 0 streams K,V (pass A); lane 1 streams Q,dO (pass B); lane 2 streams K,V (pass C)
    const int r = lane;
    __syncthreads();
    if (lane < 3) {
      const uint32_t full = smem_u32(ctrl.full[r]), empty = smem_u32(ctrl.empty[r]);
      const uint32_t base = ring + r * NST * C::KV_STAGE;
      const CUtensorMap* ma = (r == 1) ? &tmQ : &tmK;
      const CUtensorMap* mb = (r == 1) ? &tmG : &tmV;
      const int S0 = ctrl.stream_begin;
      const int total = (ctrl.stream_end - S0 + C::SR - 1) / C::SR;
      for (int st = 0; st < total; ++st) {
        if (st >= NST) mbar_wait(empty + 8u * (st % NST), (uint32_t)(((st / NST) - 1) & 1));
        const uint32_t bar = full + 8u * (st % NST);
        const uint32_t dst = base + (st % NST) * C::KV_STAGE;
        const int y = S0 + st * C::SR;
        mbar_expect_tx(bar, (uint32_t)C::KV_STAGE);
#pragma unroll
        for (int b = 0; b < C::NBOX; ++b) {
          const int x = h0 * D + 64 * b;
          tma_load_2d(dst + b * C::BOX_BYTES, ma, bar, x, y);
          tma_load_2d(dst + C::T_STAGE + b * C::BOX_BYTES, mb, bar, x, y);
        }
      }
      for (int st = max(0, total - NST); st < total; ++st)      // no TMA may be in flight at exit
        mbar_wait(full + 8u * (st % NST), (uint32_t)((st / NST) & 1));
    }
    return;
  }

  if (warp == 0) {
    int wa, wl;
    warp_windows_of_rows(off, W, R0, R1 - 1, wa, wl);
    if (lane == 0) {
      const int sa = __ldg(off + wa), ea = __ldg(off + wa + 1);
      const int sl = __ldg(off + wl), el = __ldg(off + wl + 1);
      const int ma = sa + ((ea - sa) >> 1), ml = sl + ((el - sl) >> 1);
      // fused windows: owned by the CTA whose span holds the middle row; longer ones are not ours
      const int sb = (ea - sa <= kFuseMax) ? (ma >= R0 ? sa : ea) : min(ea, R1);
      const int se = (el - sl <= kFuseMax) ? ((ml < R1) ? el : sl) : max(sl, R0);
      ctrl.wa = wa;
      ctrl.stream_begin = sb;
      ctrl.stream_end = max(se, sb);
    }
  }
  __syncthreads();
  if (warp >= nheads) return;

  const int hl = warp;
  const int S0 = ctrl.stream_begin;
  const int total = (ctrl.stream_end - S0 + C::SR - 1) / C::SR;
  RingView kv = make_ring(ring, smem_u32(ctrl.full[0]), smem_u32(ctrl.empty[0]));
  RingView qg = make_ring(ring + NST * C::KV_STAGE, smem_u32(ctrl.full[1]), smem_u32(ctrl.empty[1]));
  RingView kv2 = make_ring(ring + 2 * NST * C::KV_STAGE, smem_u32(ctrl.full[2]), smem_u32(ctrl.empty[2]));
  const size_t hcol = (size_t)(h0 + hl) * D;

  int wbase = ctrl.wa;
  int cur = __ldg(off + min(wbase + lane, W));
  int nxt = __ldg(off + min(wbase + 31 + lane, W));
  int w = wbase;
  while (w < W) {
    int i = w - wbase;
    if (i >= 31) {
      wbase += 31;
      cur = nxt;
      nxt = __ldg(off + min(wbase + 31 + lane, W));
      i = w - wbase;
    }
    const int s = __shfl_sync(0xffffffffu, cur, i), e = __shfl_sync(0xffffffffu, cur, i + 1);
    if (s >= R1) break;
    const int m = e - s;
    if (m <= 0) { ++w; continue; }
    if (m > kFuseMax) {                                   // left to the split passes
      // bounded entry (no workspace): a window that breaks the caller's promise is skipped
      if (ws != nullptr && hl == 0 && lane == 0) reinterpret_cast<volatile int*>(ws)[0] = 1;
      ++w;
      continue;
    }
    const int mid = s + (m >> 1);
    if (mid >= R1) break;
    if (mid < R0) { ++w; continue; }
    if (m <= 16) {
      // Pack the following whole short windows (owned, together <= 16 rows) into one 16-row tile, as the forward does:
      // lane j holds off[wbase+j]; one ballot finds how many consecutive windows fit, one OR-reduction the bit mask of
      // window starts inside the tile; the window ordinal of tile row r is a popcount of that mask.
      const int e_j = __shfl_down_sync(0xffffffffu, cur, 1);      // off[wbase+lane+1]
      const int mid_j = cur + ((e_j - cur) >> 1);
      const bool fits = lane >= i && lane < 31 && (e_j - s) <= 16 && mid_j < R1;
      const unsigned okm = __ballot_sync(0xffffffffu, fits) >> i;
      const int cnt = __ffs(~okm) - 1;                            // consecutive windows that fit (>= 1)
      const int rows = __shfl_sync(0xffffffffu, cur, i + cnt) - s;
      const unsigned startbit = (lane > i && lane < i + cnt) ? (1u << (cur - s)) : 0u;
      const unsigned starts = __reduce_or_sync(0xffffffffu, startbit) & 0xFFFEu;
      const int wid = (lane < rows) ? __popc(starts & ((2u << lane) - 1u)) : -1;
      w += cnt;
      const int rel = s - S0;
      ring_release_below<C::SR>(kv, rel);
      ring_release_below<C::SR>(qg, rel);
      ring_wait_upto(kv, (rel + rows - 1) / C::SR);
      ring_wait_upto(qg, (rel + rows - 1) / C::SR);
      bwd_quad_tile<MODE, T>(kv, qg, hl, rel, rows, wid, dq + hcol + (size_t)s * Ctot, dk + hcol + (size_t)s * Ctot,
                             dv + hcol + (size_t)s * Ctot, Ctot, eps);
      ring_release_below<C::SR>(kv, rel + rows);
      ring_release_below<C::SR>(qg, rel + rows);
      ring_release_below<C::SR>(kv2, rel + rows);                 // the third stream carries these rows too
      continue;
    }
    if (m <= BWD_PRECISE_MAX)
      bwd_window<MODE, true, T>(kv, qg, kv2, hl, S0, s, e, dq + hcol, dk + hcol, dv + hcol, Ctot, eps);
    else
      bwd_window<MODE, false, T>(kv, qg, kv2, hl, S0, s, e, dq + hcol, dk + hcol, dv + hcol, Ctot, eps);
    ++w;
  }
  ring_release_below<C::SR>(kv, total * C::SR);
  ring_release_below<C::SR>(qg, total * C::SR);
  ring_release_below<C::SR>(kv2, total * C::SR);
}

// ---- windows longer than kFuseMax rows: three stream-ordered passes over their pieces ----------------------------
// A piece = the intersection of such a window with one row span.  PASS 0: partial S, z of the piece -> fp32 atomics into
// the window's slot of ws_state.  PASS 1 (states complete): dq rows of the piece, partial dS, dz -> atomics into
// ws_dstate.  PASS 2: dk, dv rows.  Same tiles as the fused windows (single fp16 operand: these windows are long), one
// ring, one consumer warp per head.  A pass exits at once when the main kernel met no long window (workspace flag).
__device__ __forceinline__ float* split_slot(float* ws, int s, int H, int h) {
  return ws + kWsHeaderFloats + ((size_t)(s / (kFuseMax + 1)) * H + h) * (size_t)((D + 1) * D);
}

template <int MODE, typename T, int PASS>
__global__ void __launch_bounds__(Cfg<D>::THREADS, 2)
sla_bwd_tc_split_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB,
                        const int32_t* __restrict__ off, T* __restrict__ dq, T* __restrict__ dk, T* __restrict__ dv,
                        float* __restrict__ ws, float* __restrict__ wd, int N, int W, int H, int span, float eps) {
  constexpr bool BF16 = (MODE & 1) != 0;   // I/O dtype bf16
  constexpr int PHI = MODE >> 1;            // feature map (sla_feature_map_t)
  (void)BF16; (void)PHI;
  extern __shared__ uint8_t dyn_smem[];
  __shared__ Ctrl ctrl;
  asm volatile("griddepcontrol.launch_dependents;");
  asm volatile("griddepcontrol.wait;" ::: "memory");               // every CTA waits, so completion is transitive
  if (reinterpret_cast<const volatile int*>(ws)[0] == 0) return;   // no long window in this call
  const uint32_t ring = (smem_u32(dyn_smem) + 1023u) & ~1023u;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int R0 = blockIdx.x * span, R1 = min(R0 + span, N);
  const int h0 = blockIdx.y * NW;
  const int nheads = min(NW, H - h0);
  const int Ctot = H * D;
  if (threadIdx.x == 0) {
    for (int i = 0; i < NST; ++i) {
      mbar_init(smem_u32(&ctrl.full[0][i]), 1);
      mbar_init(smem_u32(&ctrl.empty[0][i]), nheads);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  if (warp >= NW) {   // producer: lane 0 streams the two tensors of this pass over the rows of the pieces
    __syncthreads();
    if (lane == 0) {
      const uint32_t full = smem_u32(ctrl.full[0]), empty = smem_u32(ctrl.empty[0]);
      const int S0 = ctrl.stream_begin;
      const int total = (ctrl.stream_end - S0 + C::SR - 1) / C::SR;
      for (int st = 0; st < total; ++st) {
        if (st >= NST) mbar_wait(empty + 8u * (st % NST), (uint32_t)(((st / NST) - 1) & 1));
        const uint32_t bar = full + 8u * (st % NST);
        const uint32_t dst = ring + (st % NST) * C::KV_STAGE;
        const int y = S0 + st * C::SR;
        mbar_expect_tx(bar, (uint32_t)C::KV_STAGE);
#pragma unroll
        for (int b = 0; b < C::NBOX; ++b) {
          const int x = h0 * D + 64 * b;
          tma_load_2d(dst + b * C::BOX_BYTES, &tmA, bar, x, y);
          tma_load_2d(dst + C::T_STAGE + b * C::BOX_BYTES, &tmB, bar, x, y);
        }
      }
      for (int st = max(0, total - NST); st < total; ++st)
        mbar_wait(full + 8u * (st % NST), (uint32_t)((st / NST) & 1));
    }
    return;
  }
  if (warp == 0) {
    int wa, wl;
    warp_windows_of_rows(off, W, R0, R1 - 1, wa, wl);
    if (lane == 0) {
      const int sa = __ldg(off + wa), ea = __ldg(off + wa + 1);
      const int sl = __ldg(off + wl), el = __ldg(off + wl + 1);
      // span <= kFuseMax: a long window that meets [R0,R1) holds R0 (window wa) or R1-1 (window wl)
      const bool A = ea - sa > kFuseMax, B = el - sl > kFuseMax;
      const int sb = A ? R0 : (B ? max(sl, R0) : R0);
      const int se = B ? R1 : (A ? min(ea, R1) : sb);
      ctrl.wa = wa;
      ctrl.stream_begin = sb;
      ctrl.stream_end = max(se, sb);
    }
  }
  __syncthreads();
  if (warp >= nheads) return;
  const int hl = warp, g = lane >> 2, t = lane & 3;
  const int S0 = ctrl.stream_begin;
  const int total = (ctrl.stream_end - S0 + C::SR - 1) / C::SR;
  RingView rv = make_ring(ring, smem_u32(ctrl.full[0]), smem_u32(ctrl.empty[0]));
  const size_t hcol = (size_t)(h0 + hl) * D;
  for (int w = ctrl.wa; w < W; ++w) {
    const int s = __ldg(off + w), e = __ldg(off + w + 1);
    if (s >= R1) break;
    const int m = e - s;
    if (m <= kFuseMax) continue;
    const int ps = max(s, R0), pe = min(e, R1);
    float* slot = split_slot(ws, s, H, h0 + hl);
    float* dslot = split_slot(wd, s, H, h0 + hl);
    BwdState st;
    st.clear();
    float scale = 1.f;
    if (PASS != 0) {   // the complete z of the window (pass 0 finished it): every block of the window derives the same s
#pragma unroll
      for (int nt = 0; nt < 2; ++nt)
#pragma unroll
        for (int c = 0; c < 4; ++c) st.Z[nt][c] = slot[D * D + 8 * nt + 2 * t + (c & 1)];
      scale = z_scale<2>(st.Z);
    }
    if (PASS == 0) {
      for (int r = ps; r < pe; r += 16) {
        const int nv = min(16, pe - r), rel = r - S0;
        ring_release_below<C::SR>(rv, rel);
        ring_wait_upto(rv, (rel + nv - 1) / C::SR);
        bwd_kv_tile<MODE, false>(rv, hl, rel, nv, st);
      }
#pragma unroll
      for (int nt = 0; nt < 2; ++nt)
#pragma unroll
        for (int c = 0; c < 4; ++c)      // S^T fragment: row r = g + 8 (c/2), column p = 8 nt + 2t + (c%2)
          atomicAdd(slot + (8 * nt + 2 * t + (c & 1)) * D + g + 8 * (c >> 1), st.ST[nt][c]);
      if (g == 0) {
#pragma unroll
        for (int nt = 0; nt < 2; ++nt)
#pragma unroll
          for (int c = 0; c < 2; ++c) atomicAdd(slot + D * D + 8 * nt + 2 * t + c, st.Z[nt][c]);
      }
    } else if (PASS == 1) {
#pragma unroll
      for (int nt = 0; nt < 2; ++nt)
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          st.ST[nt][c] = slot[(8 * nt + 2 * t + (c & 1)) * D + g + 8 * (c >> 1)];     // S^T[r][p] = S[p][r]
          st.Z[nt][c] = slot[D * D + 8 * nt + 2 * t + (c & 1)];
        }
      PassBOps ob;
      ob.eps = eps * scale;
      make_ops<false>(st.ST, scale, ob.num);
      transpose_ops<false>(ob.num, ob.da);
#pragma unroll
      for (int b = 0; b < 2; ++b) {
        ob.zs[b][0] = st.Z[b][0] * scale; ob.zs[b][1] = st.Z[b][1] * scale;
        to_op<false>(ob.zs[b][0], ob.zs[b][1], ob.zh[b], ob.zl[b]);
      }
      for (int r = ps; r < pe; r += 16) {
        const int nv = min(16, pe - r), rel = r - S0;
        ring_release_below<C::SR>(rv, rel);
        ring_wait_upto(rv, (rel + nv - 1) / C::SR);
        bwd_q_tile<MODE, false, T>(rv, hl, rel, nv, ob, st, dq + hcol + (size_t)r * Ctot, Ctot);
      }
#pragma unroll
      for (int nt = 0; nt < 2; ++nt)
#pragma unroll
        for (int c = 0; c < 4; ++c)      // dS^T fragment (scaled by 1/s): row r = g + 8 (c/2), column p = 8 nt + 2t + (c%2)
          atomicAdd(dslot + (8 * nt + 2 * t + (c & 1)) * D + g + 8 * (c >> 1), st.dST[nt][c]);
      if (g == 0) {
#pragma unroll
        for (int nt = 0; nt < 2; ++nt)
#pragma unroll
          for (int c = 0; c < 2; ++c) atomicAdd(dslot + D * D + 8 * nt + 2 * t + c, st.DZ[nt][c]);
      }
    } else {
      PassCOps oc;
#pragma unroll
      for (int nt = 0; nt < 2; ++nt)
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          st.dST[nt][c] = dslot[(8 * nt + 2 * t + (c & 1)) * D + g + 8 * (c >> 1)];   // dS^T[r][p]
          st.DZ[nt][c] = dslot[D * D + 8 * nt + 2 * t + (c & 1)];
        }
      make_ops<false>(st.dST, scale, oc.dv);
      transpose_ops<false>(oc.dv, oc.db);
#pragma unroll
      for (int b = 0; b < 2; ++b) { oc.dzs[b][0] = st.DZ[b][0] * scale; oc.dzs[b][1] = st.DZ[b][1] * scale; }
      for (int r = ps; r < pe; r += 16) {
        const int nv = min(16, pe - r), rel = r - S0;
        ring_release_below<C::SR>(rv, rel);
        ring_wait_upto(rv, (rel + nv - 1) / C::SR);
        bwd_kv_out_tile<MODE, false, T>(rv, hl, rel, nv, oc, dk + hcol + (size_t)r * Ctot,
                                        dv + hcol + (size_t)r * Ctot, Ctot);
      }
    }
  }
  ring_release_below<C::SR>(rv, total * C::SR);
}

template <int MODE, typename T>
cudaError_t bwd_tc_launch(const Problem& p, cudaStream_t st) {
  constexpr bool BF16 = (MODE & 1) != 0;   // I/O dtype bf16
  constexpr int PHI = MODE >> 1;            // feature map (sla_feature_map_t)
  (void)BF16; (void)PHI;
  CUtensorMap tq, tk, tv, tg;
  const int Ctot = p.H * D;
  if (!make_map(&tq, p.q, p.N, Ctot, C::SR) || !make_map(&tk, p.k, p.N, Ctot, C::SR) ||
      !make_map(&tv, p.v, p.N, Ctot, C::SR) || !make_map(&tg, p.g, p.N, Ctot, C::SR))
    return cudaErrorInvalidValue;
  auto kern = sla_bwd_tc_kernel<MODE, T>;
  static std::atomic<bool> attr_set[kMaxDevices];         // the smem opt-in is per device
  const int dev = current_device();
  if (!attr_set[dev].load(std::memory_order_acquire)) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_DYN);
    if (e != cudaSuccess) return e;
    attr_set[dev].store(true, std::memory_order_release);
  }
#ifndef SLA_BWD_SPAN
#define SLA_BWD_SPAN 64
#endif
  const int span = SLA_BWD_SPAN;   // short spans: the grid runs in many waves (dynamic balance)
  const int slabs = (p.H + NW - 1) / NW;
  // one chain of programmatic dependent launches: zeroing kernel -> main -> the three split passes
  cudaLaunchAttribute pdl[1];
  pdl[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  pdl[0].val.programmaticStreamSerializationAllowed = 1;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((p.N + span - 1) / span, slabs);
  cfg.blockDim = dim3(C::THREADS);
  cfg.dynamicSmemBytes = C::SMEM_DYN;
  cfg.stream = st;
  cfg.attrs = pdl;
  cfg.numAttrs = 1;
  cudaError_t le = cudaLaunchKernelEx(&cfg, kern, tq, tk, tv, tg, p.off, (T*)p.dq, (T*)p.dk, (T*)p.dv, p.ws_state,
                                      p.N, p.W, p.H, span, p.eps);
  if (le != cudaSuccess || p.bounded) return le;   // bounded entry: no window is left to the split passes
  // windows longer than kFuseMax rows: three passes over their pieces (each exits at once if there is none)
  auto k0 = sla_bwd_tc_split_kernel<MODE, T, 0>;
  auto k1 = sla_bwd_tc_split_kernel<MODE, T, 1>;
  auto k2 = sla_bwd_tc_split_kernel<MODE, T, 2>;
  static std::atomic<bool> attr2_set[kMaxDevices];
  if (!attr2_set[dev].load(std::memory_order_acquire)) {
    cudaError_t e = cudaFuncSetAttribute(k0, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_DYN);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k1, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_DYN);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k2, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_DYN);
    if (e != cudaSuccess) return e;
    attr2_set[dev].store(true, std::memory_order_release);
  }
  const int span2 = kFuseMax / 16 * 16;                    // the largest span the split passes handle: few pieces per window (few atomics
                                                           // per slot) and few blocks to start and retire when there is no long window
  cfg.gridDim = dim3((p.N + span2 - 1) / span2, slabs);
  le = cudaLaunchKernelEx(&cfg, k0, tk, tv, p.off, (T*)p.dq, (T*)p.dk, (T*)p.dv, p.ws_state, p.ws_dstate, p.N, p.W,
                          p.H, span2, p.eps);
  if (le == cudaSuccess)
    le = cudaLaunchKernelEx(&cfg, k1, tq, tg, p.off, (T*)p.dq, (T*)p.dk, (T*)p.dv, p.ws_state, p.ws_dstate, p.N, p.W,
                            p.H, span2, p.eps);
  if (le == cudaSuccess)
    le = cudaLaunchKernelEx(&cfg, k2, tk, tv, p.off, (T*)p.dq, (T*)p.dk, (T*)p.dv, p.ws_state, p.ws_dstate, p.N, p.W,
                            p.H, span2, p.eps);
  return le;
}

}  // namespace

bool backward_tc_supported(const Problem& p, int dt) {
  if (dt != SLA_F16 && dt != SLA_BF16) return false;
  if ((p.d != 16 && p.d != 32) || (p.H * p.d) % 64 != 0) return false;     // d_h = 32: sla_bwd_tc32.cu
  return encode_fn() != nullptr;
}

// Fused windows (<= kFuseMax rows) by sla_bwd_tc_kernel; longer windows by the three sla_bwd_tc_split_kernel passes
// (they exit at once unless the first kernel raised the workspace flag).
cudaError_t launch_backward_tc(const Problem& p, int dt, cudaStream_t st) {
  if (p.d == 32) return launch_backward_tc32(p, dt, st);
  // MODE = (bf16 ? 1 : 0) | (feature map << 1)
  const bool relu = p.phi == SLA_PHI_RELU;
  if (dt == SLA_F16) return relu ? bwd_tc_launch<2, __half>(p, st) : bwd_tc_launch<0, __half>(p, st);
  return relu ? bwd_tc_launch<3, __nv_bfloat16>(p, st) : bwd_tc_launch<1, __nv_bfloat16>(p, st);
}

}  // namespace sla
