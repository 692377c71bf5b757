// sla_bwd_tc32.cu -- SLA backward for fp16 / bf16 I/O, d_h = 32, both feature maps, on the tensor cores.
//
// The d_h = 16 kernel (sla_bwd_tc.cu) written out for a head of KS = d_h/16 column groups: the same skeleton
// (equal row spans per CTA, three TMA + mbarrier rings, one consumer warp per head, mma.sync m16n8k16 with fp32
// accumulation, window state in registers), the same three passes per window and the same gradients of Eq. 3
// (reading A14):
//   pass A (K,V):    S = sum_j b_j^T v_j (kept as S^T fragments), z = sum_j b_j
//   pass B (Q,dO):   num = a S, den = a.z, dnum = g/den, dden = -(g.o)/den
//                    dq = (dnum S^T + dden z) * phi'(q);  dS += a^T dnum;  dz += dden a
//   pass C (K,V):    dv = b dS,  dk = (v dS^T + dz) * phi'(k)
// A 32 x 32 state is four times the registers of a 16 x 16 one (S^T, dS^T, z, dz: 96 fp32 per lane), so one
// CTA of 8 head warps is resident per SM; short windows are not packed into shared tiles here (the d_h = 32 workload,
// BASELINE.json config 2, has few rows in them).  Windows longer than kFuseMax rows go through three split passes
// with their states in the fp32 workspace, as in the d_h = 16 file.
//
// Fragment conventions (g = lane/4, t = lane%4; c = accumulator register 0..3: row g (c<2) / g+8 (c>=2), column
// 2t + (c&1) of an 8-wide tile): a 32-wide matrix is KS = 2 row tiles of 16 by NT = 4 column tiles of 8:
//   X[mt][nt][c] = X(16 mt + g + 8 (c/2), 8 nt + 2t + (c&1)).
#include <cuda.h>

#include <atomic>

#include "sla_internal.cuh"

namespace sla {
namespace {

constexpr int NW = 8;     // consumer warps = heads per slab
constexpr int NST = 2;    // ring stages per stream
constexpr int BWD_PRECISE_MAX = 32;   // windows up to this length use split (hi + lo) fp16 operands

template <int DD> struct Cfg {
  static constexpr int SR = 32;                           // rows per ring stage
  static constexpr int NBOX = NW * DD / 64;               // 128-byte column boxes per slab row
  static constexpr int BOX_BYTES = SR * 128;
  static constexpr int T_STAGE = NBOX * BOX_BYTES;        // one tensor's stage (16 KB at d_h = 32)
  static constexpr int KV_STAGE = 2 * T_STAGE;            // every ring stage holds two tensors
  static constexpr int RING_BYTES = 3 * NST * KV_STAGE;   // K,V | Q,dO | K,V again
  static constexpr int SMEM_DYN = RING_BYTES + 1024;
  static constexpr int THREADS = (NW + 1) * 32;
};

#include "sla_tc_common.cuh"

constexpr int D = 32;
constexpr int KS = D / 16;   // 16-wide column groups of a head = k-steps of a contraction over channels
constexpr int NT = D / 8;    // 8-wide column tiles of a head
using C = Cfg<D>;

// Only the transposed forms S^T and dS^T are accumulated: the operands that need S and dS themselves are the 8 x 8
// block transposes (movmatrix) of the operands built from S^T and dS^T (make_pass_b_ops / make_pass_c_ops).
struct BwdState {
  float ST[KS][NT][4];    // S^T : rows r, columns p
  float Z[NT][4];         // z[p] in columns p (same in every row)
  float dST[KS][NT][4];   // dS^T (scaled by 1/s)
  float DZ[NT][4];        // dz   (scaled by 1/s)
  __device__ __forceinline__ void clear() {
#pragma unroll
    for (int a = 0; a < KS; ++a)
#pragma unroll
      for (int b = 0; b < NT; ++b)
#pragma unroll
        for (int c = 0; c < 4; ++c) { ST[a][b][c] = 0.f; dST[a][b][c] = 0.f; }
#pragma unroll
    for (int b = 0; b < NT; ++b)
#pragma unroll
      for (int c = 0; c < 4; ++c) { Z[b][c] = 0.f; DZ[b][c] = 0.f; }
  }
};

// B operands of Y = A X^T-style products, built from an accumulator X[mt][nt][c] that holds the matrix with the
// OUTPUT index in its rows and the CONTRACTION index in its columns: for output tile n (8 columns) and k-step ks,
//   op[n][ks][b] = pack(X[n/2][2 ks + b][2 (n%2)], X[n/2][2 ks + b][2 (n%2) + 1]) * scale     (b = k rows 0-7 / 8-15)
struct Ops { uint32_t hi[NT][KS][2], lo[NT][KS][2]; };

template <bool PRECISE>
__device__ __forceinline__ void to_op(float x0, float x1, uint32_t& hi, uint32_t& lo) {
  if (PRECISE) split_h2(x0, x1, hi, lo);
  else { hi = pack_h2(x0, x1); lo = 0u; }
}
template <bool PRECISE>
__device__ __forceinline__ void make_ops(const float (&X)[KS][NT][4], float scale, Ops& o) {
#pragma unroll
  for (int n = 0; n < NT; ++n)
#pragma unroll
    for (int ks = 0; ks < KS; ++ks)
#pragma unroll
      for (int b = 0; b < 2; ++b)
        to_op<PRECISE>(X[n / 2][2 * ks + b][2 * (n & 1)] * scale, X[n / 2][2 * ks + b][2 * (n & 1) + 1] * scale,
                       o.hi[n][ks][b], o.lo[n][ks][b]);
}

__device__ __forceinline__ uint32_t movm_t(uint32_t x) {   // transpose of one 8x8 block of 16-bit elements
  uint32_t y;
  asm volatile("movmatrix.sync.aligned.m8n8.trans.b16 %0, %1;" : "=r"(y) : "r"(x));
  return y;
}
// Operands of the transposed matrix: o holds the 8 x 8 blocks (output block n, contraction block 2 ks + b) of X; the
// same blocks of X^T are the transposes of the blocks (2 ks + b, n) of X.
template <bool PRECISE>
__device__ __forceinline__ void transpose_ops(const Ops& o, Ops& t) {
#pragma unroll
  for (int n = 0; n < NT; ++n)
#pragma unroll
    for (int ks = 0; ks < KS; ++ks)
#pragma unroll
      for (int b = 0; b < 2; ++b) {
        const int m = 2 * ks + b;                      // contraction block of t = output block of o
        t.hi[n][ks][b] = movm_t(o.hi[m][n >> 1][n & 1]);
        t.lo[n][ks][b] = PRECISE ? movm_t(o.lo[m][n >> 1][n & 1]) : 0u;
      }
}

// phi of a packed pair in fp32 (a) and its derivative factor: elu+1: (x > 0 ? 1 : phi(x)); ReLU: [x > 0]
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
// 16-byte chunk of column group ks of head hl inside the slab row (a head is D/8 chunks)
__device__ __forceinline__ int head_chunk(int hl, int ks, int csel) { return hl * (D / 8) + 2 * ks + csel; }

// ---- pass A: one 16-row K/V tile -> S^T, z ----------------------------------------------------------
template <int MODE, bool PRECISE>
__device__ __forceinline__ void bwd_kv_tile(const RingView& rv, int hl, int rel0, int nvalid, BwdState& s) {
  constexpr bool BF16 = (MODE & 1) != 0;   // I/O dtype bf16
  constexpr int PHI = MODE >> 1;            // feature map (sla_feature_map_t)
  (void)BF16; (void)PHI;
  const int t = threadIdx.x & 3;
  int trow, csel;
  lane_pattern(nvalid, trow, csel);
  // transposed loads: kr[ks][i] = K[j = 2t,2t+1 (+8 for i>=2)][p = 16 ks + g (+8 for odd i)], same for vr with r
  uint32_t bh[KS][4], bl[KS][4], vr[KS][4];
#pragma unroll
  for (int ks = 0; ks < KS; ++ks) {
    uint32_t kr[4];
    ldsm_x4_t(ring_addr<D>(rv, C::KV_STAGE, 0, rel0 + trow, head_chunk(hl, ks, csel)), kr);
    ldsm_x4_t(ring_addr<D>(rv, C::KV_STAGE, C::T_STAGE, rel0 + trow, head_chunk(hl, ks, csel)), vr[ks]);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const int j0 = 2 * t + 8 * (i >> 1);
      if (PRECISE) {
        const float2 x = unpack2<BF16>(kr[i]);
        const float b0 = (j0 < nvalid) ? phi_fast<PHI>(x.x) : 0.f;
        const float b1 = (j0 + 1 < nvalid) ? phi_fast<PHI>(x.y) : 0.f;
        to_op<true>(b0, b1, bh[ks][i], bl[ks][i]);
      } else {   // long window: phi in fp16x2 (the operand is a single fp16 anyway), rows beyond the window zeroed
        bh[ks][i] = phi_h2<BF16, PHI>(kr[i]);
        if (nvalid < 16) bh[ks][i] &= pair_mask(j0, nvalid);
        bl[ks][i] = 0u;
      }
    }
    if (BF16) {
#pragma unroll
      for (int i = 0; i < 4; ++i) { const float2 x = unpack2<true>(vr[ks][i]); vr[ks][i] = pack_h2(x.x, x.y); }
    }
  }
  const uint32_t ones = 0x3C003C00u;
#pragma unroll
  for (int nt = 0; nt < NT; ++nt) {
    const int kc = nt >> 1, hf = nt & 1;      // column tile nt = half hf of column group kc
    mma16816(s.Z[nt], ones, ones, ones, ones, bh[kc][hf], bh[kc][2 + hf]);
    if (PRECISE) mma16816(s.Z[nt], ones, ones, ones, ones, bl[kc][hf], bl[kc][2 + hf]);
#pragma unroll
    for (int mt = 0; mt < KS; ++mt) {
      // S^T (rows r of group mt, cols p of tile nt): A = V^T, B = phi(K)
      mma16816(s.ST[mt][nt], vr[mt][0], vr[mt][1], vr[mt][2], vr[mt][3], bh[kc][hf], bh[kc][2 + hf]);
      if (PRECISE) mma16816(s.ST[mt][nt], vr[mt][0], vr[mt][1], vr[mt][2], vr[mt][3], bl[kc][hf], bl[kc][2 + hf]);
    }
  }
}

struct PassBOps {
  Ops num;                   // from S^T: B operand of num = a S
  Ops da;                    // from S  : B operand of da = dnum S^T
  uint32_t zh[KS][2], zl[KS][2];   // z as B operand of den
  float zs[NT][2];           // scaled z in columns p = 8 np + 2t + c
  float eps;                 // epsilon of the denominator on the scale of the operands (eps * s); 0 for elu+1
};

// ---- pass B: one 16-row Q/dO tile -> dq rows, dS^T, dz accumulators ----------------------------------
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
  const int perm[4] = {0, 2, 1, 3};   // ldmatrix register order -> A-fragment order (a0..a3)
  // A fragments of column group ks: 0: (row g, cols 2t..), 1: (row g+8, cols 2t..), 2: (row g, cols 8+2t..), 3: (row g+8, 8+2t..)
  uint32_t ah[KS][4], al[KS][4], dph2[KS][4], graw[KS][4];
  float2 dph[KS][4], gv[KS][4];
#pragma unroll
  for (int ks = 0; ks < KS; ++ks) {
    uint32_t qn[4], gn[4];
    ldsm_x4(ring_addr<D>(rv, C::KV_STAGE, 0, rel0 + trow, head_chunk(hl, ks, csel)), qn);
    ldsm_x4(ring_addr<D>(rv, C::KV_STAGE, C::T_STAGE, rel0 + trow, head_chunk(hl, ks, csel)), gn);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      if (PRECISE) {
        float2 a;
        phi_pair<MODE>(qn[perm[i]], a, dph[ks][i]);
        to_op<true>(a.x, a.y, ah[ks][i], al[ks][i]);
      } else {
        phi_dphi_h2<BF16, PHI>(qn[perm[i]], ah[ks][i], dph2[ks][i]);
        al[ks][i] = 0u;
      }
      graw[ks][i] = gn[perm[i]];
      gv[ks][i] = unpack2<BF16>(gn[perm[i]]);
    }
  }
  float num[NT][4], den[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
  for (int ks = 0; ks < KS; ++ks) mma3<PRECISE>(den, ah[ks], al[ks], op.zh[ks][0], op.zh[ks][1], op.zl[ks][0], op.zl[ks][1]);
#pragma unroll
  for (int n = 0; n < NT; ++n) {
#pragma unroll
    for (int c = 0; c < 4; ++c) num[n][c] = 0.f;
#pragma unroll
    for (int ks = 0; ks < KS; ++ks)
      mma3<PRECISE>(num[n], ah[ks], al[ks], op.num.hi[n][ks][0], op.num.hi[n][ks][1], op.num.lo[n][ks][0], op.num.lo[n][ks][1]);
  }
  const float inv0 = fast_rcp(PHI ? den[0] + op.eps : den[0]), inv1 = fast_rcp(PHI ? den[2] + op.eps : den[2]);   // rows g, g+8
  // g.o per row: this lane holds columns 8n + 2t, +1 of rows g and g+8 for every tile n
  float go0 = 0.f, go1 = 0.f;
#pragma unroll
  for (int n = 0; n < NT; ++n) {
    const float2 g0 = gv[n >> 1][2 * (n & 1)], g1 = gv[n >> 1][2 * (n & 1) + 1];
    go0 += g0.x * num[n][0] + g0.y * num[n][1];
    go1 += g1.x * num[n][2] + g1.y * num[n][3];
  }
  go0 += __shfl_xor_sync(0xffffffffu, go0, 1); go0 += __shfl_xor_sync(0xffffffffu, go0, 2);
  go1 += __shfl_xor_sync(0xffffffffu, go1, 1); go1 += __shfl_xor_sync(0xffffffffu, go1, 2);
  const float dden0 = -(go0 * inv0) * inv0, dden1 = -(go1 * inv1) * inv1;   // o = num*inv
  // ReLU: rows whose denominator is almost eps alone make g/den and dden huge; rescale the tile by a power of two
  float gmax = 0.f;
  if (PHI) {
#pragma unroll
    for (int ks = 0; ks < KS; ++ks)
#pragma unroll
      for (int i = 0; i < 4; ++i)
        gmax = fmaxf(gmax, fmaxf(fabsf(gv[ks][i].x), fabsf(gv[ks][i].y)) * ((i & 1) ? inv1 : inv0));
    gmax = fmaxf(gmax, fmaxf(fabsf(dden0), fabsf(dden1)));
  }
  const int ksh = tile_shift<PHI>(gmax);
  const float dn = pow2f(-ksh), up = pow2f(ksh);        // both 1 unless ReLU and an ill-conditioned row
  // dnum as A fragments (rows g / g+8 scaled by their 1/den)
  uint32_t dh[KS][4], dl[KS][4];
#pragma unroll
  for (int ks = 0; ks < KS; ++ks)
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const float iv = ((i & 1) ? inv1 : inv0) * dn;
      if (PRECISE || BF16 || PHI)
        to_op<PRECISE>(sat_h<PHI>(gv[ks][i].x * iv), sat_h<PHI>(gv[ks][i].y * iv), dh[ks][i], dl[ks][i]);
      else { dh[ks][i] = hmul2_u32(graw[ks][i], pack_h2(iv, iv)); dl[ks][i] = 0u; }
    }
  // da = dnum S^T + dden z ; dq = da * phi'(q)
#pragma unroll
  for (int np = 0; np < NT; ++np) {
    float da[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
    for (int ks = 0; ks < KS; ++ks)
      mma3<PRECISE>(da, dh[ks], dl[ks], op.da.hi[np][ks][0], op.da.hi[np][ks][1], op.da.lo[np][ks][0], op.da.lo[np][ks][1]);
    // C fragment (np): c0,c1 = (row g, p = 8np+2t,+1) <-> A index 2 (np%2) of group np/2 ; c2,c3 = row g+8 <-> A index + 1
    if (PHI) { da[0] *= up; da[1] *= up; da[2] *= up; da[3] *= up; }
    const float q0 = da[0] + dden0 * op.zs[np][0], q1 = da[1] + dden0 * op.zs[np][1];
    const float q2 = da[2] + dden1 * op.zs[np][0], q3 = da[3] + dden1 * op.zs[np][1];
    uint32_t* p0 = reinterpret_cast<uint32_t*>(dq_rows + (size_t)g * C_total + 8 * np + 2 * t);
    uint32_t* p1 = reinterpret_cast<uint32_t*>(dq_rows + (size_t)(g + 8) * C_total + 8 * np + 2 * t);
    const int kg = np >> 1, ai = 2 * (np & 1);
    if (PRECISE) {
      if (g < nvalid) *p0 = pack_out<BF16>(q0 * dph[kg][ai].x, q1 * dph[kg][ai].y);
      if (g + 8 < nvalid) *p1 = pack_out<BF16>(q2 * dph[kg][ai + 1].x, q3 * dph[kg][ai + 1].y);
    } else {
      if (g < nvalid) *p0 = pack_out_times_h2<BF16, PHI != 0>(q0, q1, dph2[kg][ai]);
      if (g + 8 < nvalid) *p1 = pack_out_times_h2<BF16, PHI != 0>(q2, q3, dph2[kg][ai + 1]);
    }
  }
  // ---- transposed operands (contraction over the rows i of the tile) ----
  // 1/den and dden of rows 2t, 2t+1, 2t+8, 2t+9 live in the lanes whose g equals that row
  const int l0 = 4 * (2 * t), l1 = 4 * (2 * t + 1);
  const float ir0 = __shfl_sync(0xffffffffu, inv0, l0), ir1 = __shfl_sync(0xffffffffu, inv0, l1);
  const float ir2 = __shfl_sync(0xffffffffu, inv1, l0), ir3 = __shfl_sync(0xffffffffu, inv1, l1);
  const float dd0 = __shfl_sync(0xffffffffu, dden0, l0), dd1 = __shfl_sync(0xffffffffu, dden0, l1);
  const float dd2 = __shfl_sync(0xffffffffu, dden1, l0), dd3 = __shfl_sync(0xffffffffu, dden1, l1);
  uint32_t uh[KS][4], ul[KS][4], th[KS][4], tl[KS][4];
#pragma unroll
  for (int ks = 0; ks < KS; ++ks) {
    // qt[i] = Q[i' = 2t,2t+1 (+8 for i>=2)][p = 16 ks + g (+8 for odd i)] ; gt[i] likewise with r
    uint32_t qt[4], gt[4];
    ldsm_x4_t(ring_addr<D>(rv, C::KV_STAGE, 0, rel0 + trow, head_chunk(hl, ks, csel)), qt);
    ldsm_x4_t(ring_addr<D>(rv, C::KV_STAGE, C::T_STAGE, rel0 + trow, head_chunk(hl, ks, csel)), gt);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const int i0 = 2 * t + 8 * (i >> 1);
      const float s0 = ((i >> 1) ? ir2 : ir0) * dn, s1 = ((i >> 1) ? ir3 : ir1) * dn;   // dn = 1 unless ReLU
      if (PRECISE) {
        const float2 x = unpack2<BF16>(qt[i]);
        const float a0 = (i0 < nvalid) ? phi_fast<PHI>(x.x) : 0.f;       // rows beyond the window contribute nothing
        const float a1 = (i0 + 1 < nvalid) ? phi_fast<PHI>(x.y) : 0.f;
        to_op<true>(sat_h<PHI>(a0 * up), sat_h<PHI>(a1 * up), uh[ks][i], ul[ks][i]);
      } else {
        uh[ks][i] = phi_h2<BF16, PHI>(qt[i]);
        if (nvalid < 16) uh[ks][i] &= pair_mask(i0, nvalid);
        if (PHI) uh[ks][i] = hmul2_u32(uh[ks][i], pack_h2(up, up));
        ul[ks][i] = 0u;
      }
      if (PRECISE || BF16 || PHI) {
        const float2 gg = unpack2<BF16>(gt[i]);
        to_op<PRECISE>(sat_h<PHI>(gg.x * s0), sat_h<PHI>(gg.y * s1), th[ks][i], tl[ks][i]);
      } else {
        th[ks][i] = hmul2_u32(gt[i], pack_h2(s0, s1));
        tl[ks][i] = 0u;
      }
    }
  }
  uint32_t ddh[2], ddl[2];
  to_op<PRECISE>(sat_h<PHI>(dd0 * dn), sat_h<PHI>(dd1 * dn), ddh[0], ddl[0]);
  to_op<PRECISE>(sat_h<PHI>(dd2 * dn), sat_h<PHI>(dd3 * dn), ddh[1], ddl[1]);
  const uint32_t dda_h[4] = {ddh[0], ddh[0], ddh[1], ddh[1]}, dda_l[4] = {ddl[0], ddl[0], ddl[1], ddl[1]};
#pragma unroll
  for (int nt = 0; nt < NT; ++nt) {
    const int kc = nt >> 1, hf = nt & 1;
    // dz[p] = sum_i dden_i a_i[p]: A rows all equal to dden over i, B = a tile nt
    mma3<PRECISE>(s.DZ[nt], dda_h, dda_l, uh[kc][hf], uh[kc][2 + hf], ul[kc][hf], ul[kc][2 + hf]);
#pragma unroll
    for (int mt = 0; mt < KS; ++mt) {
      // dS^T (rows r of group mt, cols p of tile nt): A = dnum^T, B = a
      mma3<PRECISE>(s.dST[mt][nt], th[mt], tl[mt], uh[kc][hf], uh[kc][2 + hf], ul[kc][hf], ul[kc][2 + hf]);
    }
  }
}

struct PassCOps {
  Ops dv;                // from dS^T: B operand of dv = b dS
  Ops db;                // from dS  : B operand of db = v dS^T
  float dzs[NT][2];      // dz in columns p = 8 np + 2t + c
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
  const int perm[4] = {0, 2, 1, 3};
  uint32_t bh[KS][4], bl[KS][4], vh[KS][4], dph2[KS][4];
  float2 dph[KS][4];
#pragma unroll
  for (int ks = 0; ks < KS; ++ks) {
    uint32_t kn[4], vn[4];
    ldsm_x4(ring_addr<D>(rv, C::KV_STAGE, 0, rel0 + trow, head_chunk(hl, ks, csel)), kn);
    ldsm_x4(ring_addr<D>(rv, C::KV_STAGE, C::T_STAGE, rel0 + trow, head_chunk(hl, ks, csel)), vn);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      if (PRECISE) {
        float2 b;
        phi_pair<MODE>(kn[perm[i]], b, dph[ks][i]);
        to_op<true>(b.x, b.y, bh[ks][i], bl[ks][i]);
      } else {
        phi_dphi_h2<BF16, PHI>(kn[perm[i]], bh[ks][i], dph2[ks][i]);
        bl[ks][i] = 0u;
      }
      if (BF16) { const float2 x = unpack2<true>(vn[perm[i]]); vh[ks][i] = pack_h2(x.x, x.y); }
      else vh[ks][i] = vn[perm[i]];
    }
  }
#pragma unroll
  for (int n = 0; n < NT; ++n) {
    float dv[4] = {0.f, 0.f, 0.f, 0.f}, db[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
    for (int ks = 0; ks < KS; ++ks) {
      mma3<PRECISE>(dv, bh[ks], bl[ks], op.dv.hi[n][ks][0], op.dv.hi[n][ks][1], op.dv.lo[n][ks][0], op.dv.lo[n][ks][1]);
      mma16816(db, vh[ks][0], vh[ks][1], vh[ks][2], vh[ks][3], op.db.hi[n][ks][0], op.db.hi[n][ks][1]);
      if (PRECISE)   // v is exact: only the operand built from dS has a residual
        mma16816(db, vh[ks][0], vh[ks][1], vh[ks][2], vh[ks][3], op.db.lo[n][ks][0], op.db.lo[n][ks][1]);
    }
    const float k0 = db[0] + op.dzs[n][0], k1 = db[1] + op.dzs[n][1];
    const float k2 = db[2] + op.dzs[n][0], k3 = db[3] + op.dzs[n][1];
    const size_t o0 = (size_t)g * C_total + 8 * n + 2 * t, o1 = (size_t)(g + 8) * C_total + 8 * n + 2 * t;
    const int kg = n >> 1, ai = 2 * (n & 1);
    if (g < nvalid) {
      *reinterpret_cast<uint32_t*>(dv_rows + o0) = pack_out<BF16>(dv[0], dv[1]);
      *reinterpret_cast<uint32_t*>(dk_rows + o0) = PRECISE ? pack_out<BF16>(k0 * dph[kg][ai].x, k1 * dph[kg][ai].y)
                                                           : pack_out_times_h2<BF16, PHI != 0>(k0, k1, dph2[kg][ai]);
    }
    if (g + 8 < nvalid) {
      *reinterpret_cast<uint32_t*>(dv_rows + o1) = pack_out<BF16>(dv[2], dv[3]);
      *reinterpret_cast<uint32_t*>(dk_rows + o1) = PRECISE ? pack_out<BF16>(k2 * dph[kg][ai + 1].x, k3 * dph[kg][ai + 1].y)
                                                           : pack_out_times_h2<BF16, PHI != 0>(k2, k3, dph2[kg][ai + 1]);
    }
  }
}

// operands of pass B from the complete state, and of pass C from the complete dS, dz (both on the window's scale)
template <bool PRECISE>
__device__ __forceinline__ void make_pass_b_ops(const BwdState& st, float scale, float eps, PassBOps& ob) {
  ob.eps = eps * scale;
  make_ops<PRECISE>(st.ST, scale, ob.num);
  transpose_ops<PRECISE>(ob.num, ob.da);
#pragma unroll
  for (int n = 0; n < NT; ++n) { ob.zs[n][0] = st.Z[n][0] * scale; ob.zs[n][1] = st.Z[n][1] * scale; }
#pragma unroll
  for (int ks = 0; ks < KS; ++ks)
#pragma unroll
    for (int b = 0; b < 2; ++b)
      to_op<PRECISE>(ob.zs[2 * ks + b][0], ob.zs[2 * ks + b][1], ob.zh[ks][b], ob.zl[ks][b]);
}
template <bool PRECISE>
__device__ __forceinline__ void make_pass_c_ops(const BwdState& st, float scale, PassCOps& oc) {
  make_ops<PRECISE>(st.dST, scale, oc.dv);
  transpose_ops<PRECISE>(oc.dv, oc.db);
#pragma unroll
  for (int n = 0; n < NT; ++n) { oc.dzs[n][0] = st.DZ[n][0] * scale; oc.dzs[n][1] = st.DZ[n][1] * scale; }
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
  const float scale = z_scale<NT>(st.Z);                  // s: largest z of the window -> [1, 2) (sla_tc_base.cuh)
  {
    PassBOps ob;
    make_pass_b_ops<PRECISE>(st, scale, eps, ob);
    for (int r = s; r < e; r += 16) {
      const int nv = min(16, e - r), rel = r - S0;
      ring_release_below<C::SR>(qg, rel);
      ring_wait_upto(qg, (rel + nv - 1) / C::SR);
      bwd_q_tile<MODE, PRECISE, T>(qg, hl, rel, nv, ob, st, dq_head + (size_t)r * Ctot, Ctot);
    }
  }
  PassCOps oc;
  make_pass_c_ops<PRECISE>(st, scale, oc);
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

// stream `total` stages of two tensors (boxes of 64 columns x SR rows) into one ring; lane-private, one lane per ring
__device__ __forceinline__ void produce_ring(uint32_t base, uint32_t full, uint32_t empty, const CUtensorMap* ma,
                                             const CUtensorMap* mb, int S0, int total, int x0) {
  for (int st = 0; st < total; ++st) {
    if (st >= NST) mbar_wait(empty + 8u * (st % NST), (uint32_t)(((st / NST) - 1) & 1));
    const uint32_t bar = full + 8u * (st % NST);
    const uint32_t dst = base + (st % NST) * C::KV_STAGE;
    const int y = S0 + st * C::SR;
    mbar_expect_tx(bar, (uint32_t)C::KV_STAGE);
#pragma unroll
    for (int b = 0; b < C::NBOX; ++b) {
      tma_load_2d(dst + b * C::BOX_BYTES, ma, bar, x0 + 64 * b, y);
      tma_load_2d(dst + C::T_STAGE + b * C::BOX_BYTES, mb, bar, x0 + 64 * b, y);
    }
  }
  for (int st = max(0, total - NST); st < total; ++st)      // no TMA may be in flight at exit
    mbar_wait(full + 8u * (st % NST), (uint32_t)((st / NST) & 1));
}

// Fused windows (<= kFuseMax rows): every CTA owns the windows whose middle row lies in its span.
template <int MODE, typename T>
__global__ void __launch_bounds__(C::THREADS, 1)
sla_bwd_tc32_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmK,
                    const __grid_constant__ CUtensorMap tmV, const __grid_constant__ CUtensorMap tmG,
                    const int32_t* __restrict__ off, T* __restrict__ dq, T* __restrict__ dk,
                    T* __restrict__ dv, float* __restrict__ ws, int N, int W, int H, int span, float eps) {
  constexpr bool BF16 = (MODE & 1) != 0;   // I/O dtype bf16
  constexpr int PHI = MODE >> 1;            // feature map (sla_feature_map_t)
  (void)BF16; (void)PHI;
  extern __shared__ uint8_t dyn_smem[];
  __shared__ Ctrl ctrl;
  // programmatic dependent launch: resident behind the previous kernel's tail; the barrier set-up runs ahead,
  // nothing that kernel may have written is touched before griddepcontrol.wait
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
    __syncthreads();
    if (lane < 3) {
      const int S0 = ctrl.stream_begin;
      produce_ring(ring + lane * NST * C::KV_STAGE, smem_u32(ctrl.full[lane]), smem_u32(ctrl.empty[lane]),
                   (lane == 1) ? &tmQ : &tmK, (lane == 1) ? &tmG : &tmV, S0,
                   (ctrl.stream_end - S0 + C::SR - 1) / C::SR, h0 * D);
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

  for (int w = ctrl.wa; w < W; ++w) {
    const int s = __ldg(off + w), e = __ldg(off + w + 1);
    if (s >= R1) break;
    const int m = e - s;
    if (m <= 0) continue;
    if (m > kFuseMax) {                                   // left to the split passes
      // bounded entry (no workspace): a window that breaks the caller's promise is skipped
      if (ws != nullptr && hl == 0 && lane == 0) reinterpret_cast<volatile int*>(ws)[0] = 1;
      continue;
    }
    const int mid = s + (m >> 1);
    if (mid >= R1) break;
    if (mid < R0) continue;
    if (m <= BWD_PRECISE_MAX)
      bwd_window<MODE, true, T>(kv, qg, kv2, hl, S0, s, e, dq + hcol, dk + hcol, dv + hcol, Ctot, eps);
    else
      bwd_window<MODE, false, T>(kv, qg, kv2, hl, S0, s, e, dq + hcol, dk + hcol, dv + hcol, Ctot, eps);
  }
  ring_release_below<C::SR>(kv, total * C::SR);
  ring_release_below<C::SR>(qg, total * C::SR);
  ring_release_below<C::SR>(kv2, total * C::SR);
}

// ---- windows longer than kFuseMax rows: three stream-ordered passes over their pieces ----------------------------
// A piece = the intersection of such a window with one row span.  PASS 0: partial S, z of the piece -> fp32 atomics into
// the window's slot of ws_state ([d+1][d]: S[p][r] at p*d + r, z[p] in row d).  PASS 1 (states complete): dq rows of
// the piece, partial dS, dz -> atomics into ws_dstate.  PASS 2: dk, dv rows.  Single fp16 operands (these windows are
// long).  A pass exits at once when the main kernel met no long window (workspace flag).
__device__ __forceinline__ float* split_slot(float* ws, int s, int H, int h) {
  return ws + kWsHeaderFloats + ((size_t)(s / (kFuseMax + 1)) * H + h) * (size_t)((D + 1) * D);
}

template <int MODE, typename T, int PASS>
__global__ void __launch_bounds__(C::THREADS, 1)
sla_bwd_tc32_split_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB,
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
      const int S0 = ctrl.stream_begin;
      produce_ring(ring, smem_u32(ctrl.full[0]), smem_u32(ctrl.empty[0]), &tmA, &tmB, S0,
                   (ctrl.stream_end - S0 + C::SR - 1) / C::SR, h0 * D);
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
      for (int nt = 0; nt < NT; ++nt)
#pragma unroll
        for (int c = 0; c < 4; ++c) st.Z[nt][c] = slot[D * D + 8 * nt + 2 * t + (c & 1)];
      scale = z_scale<NT>(st.Z);
    }
    // fragment X[mt][nt][c] <-> matrix element (row 16 mt + g + 8 (c/2), column 8 nt + 2t + (c&1))
    if (PASS == 0) {
      for (int r = ps; r < pe; r += 16) {
        const int nv = min(16, pe - r), rel = r - S0;
        ring_release_below<C::SR>(rv, rel);
        ring_wait_upto(rv, (rel + nv - 1) / C::SR);
        bwd_kv_tile<MODE, false>(rv, hl, rel, nv, st);
      }
#pragma unroll
      for (int mt = 0; mt < KS; ++mt)
#pragma unroll
        for (int nt = 0; nt < NT; ++nt)
#pragma unroll
          for (int c = 0; c < 4; ++c)      // S^T fragment: row r, column p -> S[p][r]
            atomicAdd(slot + (8 * nt + 2 * t + (c & 1)) * D + 16 * mt + g + 8 * (c >> 1), st.ST[mt][nt][c]);
      if (g == 0) {
#pragma unroll
        for (int nt = 0; nt < NT; ++nt)
#pragma unroll
          for (int c = 0; c < 2; ++c) atomicAdd(slot + D * D + 8 * nt + 2 * t + c, st.Z[nt][c]);
      }
    } else if (PASS == 1) {
#pragma unroll
      for (int mt = 0; mt < KS; ++mt)
#pragma unroll
        for (int nt = 0; nt < NT; ++nt)
#pragma unroll
          for (int c = 0; c < 4; ++c) {
            const int row = 16 * mt + g + 8 * (c >> 1), col = 8 * nt + 2 * t + (c & 1);
            st.ST[mt][nt][c] = slot[col * D + row];     // S^T[r][p] = S[p][r]
          }
#pragma unroll
      for (int nt = 0; nt < NT; ++nt)
#pragma unroll
        for (int c = 0; c < 4; ++c) st.Z[nt][c] = slot[D * D + 8 * nt + 2 * t + (c & 1)];
      PassBOps ob;
      make_pass_b_ops<false>(st, scale, eps, ob);
      for (int r = ps; r < pe; r += 16) {
        const int nv = min(16, pe - r), rel = r - S0;
        ring_release_below<C::SR>(rv, rel);
        ring_wait_upto(rv, (rel + nv - 1) / C::SR);
        bwd_q_tile<MODE, false, T>(rv, hl, rel, nv, ob, st, dq + hcol + (size_t)r * Ctot, Ctot);
      }
#pragma unroll
      for (int mt = 0; mt < KS; ++mt)
#pragma unroll
        for (int nt = 0; nt < NT; ++nt)
#pragma unroll
          for (int c = 0; c < 4; ++c)      // dS^T fragment (scaled by 1/s): row r, column p -> dS[p][r]
            atomicAdd(dslot + (8 * nt + 2 * t + (c & 1)) * D + 16 * mt + g + 8 * (c >> 1), st.dST[mt][nt][c]);
      if (g == 0) {
#pragma unroll
        for (int nt = 0; nt < NT; ++nt)
#pragma unroll
          for (int c = 0; c < 2; ++c) atomicAdd(dslot + D * D + 8 * nt + 2 * t + c, st.DZ[nt][c]);
      }
    } else {
#pragma unroll
      for (int mt = 0; mt < KS; ++mt)
#pragma unroll
        for (int nt = 0; nt < NT; ++nt)
#pragma unroll
          for (int c = 0; c < 4; ++c) {
            const int row = 16 * mt + g + 8 * (c >> 1), col = 8 * nt + 2 * t + (c & 1);
            st.dST[mt][nt][c] = dslot[col * D + row];   // dS^T[r][p]
          }
#pragma unroll
      for (int nt = 0; nt < NT; ++nt)
#pragma unroll
        for (int c = 0; c < 4; ++c) st.DZ[nt][c] = dslot[D * D + 8 * nt + 2 * t + (c & 1)];
      PassCOps oc;
      make_pass_c_ops<false>(st, scale, oc);
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
cudaError_t bwd_tc32_launch(const Problem& p, cudaStream_t st) {
  constexpr bool BF16 = (MODE & 1) != 0;   // I/O dtype bf16
  constexpr int PHI = MODE >> 1;            // feature map (sla_feature_map_t)
  (void)BF16; (void)PHI;
  CUtensorMap tq, tk, tv, tg;
  const int Ctot = p.H * D;
  if (!make_map(&tq, p.q, p.N, Ctot, C::SR) || !make_map(&tk, p.k, p.N, Ctot, C::SR) ||
      !make_map(&tv, p.v, p.N, Ctot, C::SR) || !make_map(&tg, p.g, p.N, Ctot, C::SR))
    return cudaErrorInvalidValue;
  auto kern = sla_bwd_tc32_kernel<MODE, T>;
  auto k0 = sla_bwd_tc32_split_kernel<MODE, T, 0>;
  auto k1 = sla_bwd_tc32_split_kernel<MODE, T, 1>;
  auto k2 = sla_bwd_tc32_split_kernel<MODE, T, 2>;
  static std::atomic<bool> attr_set[kMaxDevices];         // the smem opt-in is per device
  const int dev = current_device();
  if (!attr_set[dev].load(std::memory_order_acquire)) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_DYN);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k0, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_DYN);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k1, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_DYN);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k2, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_DYN);
    if (e != cudaSuccess) return e;
    attr_set[dev].store(true, std::memory_order_release);
  }
#ifndef SLA_BWD32_SPAN
#define SLA_BWD32_SPAN 64
#endif
  const int span = SLA_BWD32_SPAN;
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
  const int span2 = kFuseMax / 16 * 16;            // the largest span the split passes handle: 33 x 32 atomics per piece and head
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

cudaError_t launch_backward_tc32(const Problem& p, int dt, cudaStream_t st) {
  // MODE = (bf16 ? 1 : 0) | (feature map << 1)
  const bool relu = p.phi == SLA_PHI_RELU;
  if (dt == SLA_F16) return relu ? bwd_tc32_launch<2, __half>(p, st) : bwd_tc32_launch<0, __half>(p, st);
  return relu ? bwd_tc32_launch<3, __nv_bfloat16>(p, st) : bwd_tc32_launch<1, __nv_bfloat16>(p, st);
}

}  // namespace sla
