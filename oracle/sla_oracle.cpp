// sla_oracle.cpp -- CPU ORACLE for Scattered Linear Attention (ScatterFormer, arxiv 2401.00912).
//
// THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
// cpu_baseline / --impl reference legs may load it.  It shares no code, header, table or helper with
// the CUDA path under paper_2401_00912_b200/csrc/, and neither includes the other.
//
// What it computes is the plain definition, written out as loops in fp64 (the method reaches exactly
// this result, up to rounding order, so the oracle is the definition and not the chunk algorithm):
//
//   Eq. 2  SLA(Q,K,V) = Concat_j LA(Q^j, K^j, V^j)           -- windows are independent
//   Eq. 3  O^j = phi(Q) sum_i phi(K_i)^T V_i / ( phi(Q) sum_i phi(K_i)^T )
//   state convention: S = sum_i phi(k_i)^T v_i in R^{d x d}, row vector o = q S
//   flat window-sorted layout: voxels of window w are rows off[w] .. off[w+1]-1
//   heads: Eq. 3 applied per head with its own d_h x d_h state.
//
// Readings of points the paper leaves open:
//   A1 phi(x) = elu(x)+1  (Eq. 3's defining sentence cites [17] = Katharopoulos et al.)
//   A2 no epsilon in the denominator; A3 no 1/sqrt(d); A4 non-causal (sum over the whole window);
//   A6 the denominator is one scalar per (voxel, head); A7 empty windows allowed and skipped.
//
//   A15 second feature map, kind = 1: phi(x) = max(x, 0) with an epsilon added to the denominator,
//       o_i = phi(q_i) S / (phi(q_i) . z + eps).  Table 7's default-valued row is labelled "Efficient Attn [3]"
//       (PAPER.md:277, 296), a ReLU kernel; the paper prints neither the map nor an epsilon, and without one the
//       denominator can be exactly 0 (every phi(q_i)[p] phi(k_j)[p] = 0), so eps is an argument (default 1e-6 in
//       the callers).  kind = 0 with eps = 0 is reading A1/A2 above, unchanged.
//
// Backward: the paper is silent; these are the analytic derivatives of Eq. 3 under the readings above
// (SURVEY.md §8c), pinned in tests/test_oracle_pins.py by finite differences, torch autograd on the
// quadratic form, and the identities P6.
//
// The ReLU map's pins (same file, "relu" tests): quadratic form with eps by brute force, homogeneity in q and in all
// k of a window at eps = 0, the closed form o(eps) = o(0) den/(den+eps), length-1 windows, a hand-derived d = 2
// example (tests/golden/sla_golden_relu_d2.txt), autograd on the quadratic form and finite differences.
//
// Pins (tests/test_oracle_pins.py): P1 brute-force quadratic form, P2 closed forms, P3 invariants,
// P4 padded masked group attention, P5 golden example tests/golden/sla_golden_d2.txt, P6 gradient
// identities, P7 finite differences.  Nothing here is "parity unpinned".
//
// Build: g++ -O2 -std=c++17 -shared -fPIC -pthread oracle/sla_oracle.cpp -o oracle/libsla_oracle.so

#include <cmath>
#include <cstdint>
#include <thread>
#include <vector>
#include <algorithm>

namespace {

// kind 0: elu(x)+1 (reading A1); kind 1: max(x, 0) (reading A15) -- and their derivatives
inline double phi(double x, int kind) { return kind == 1 ? (x > 0.0 ? x : 0.0) : (x > 0.0 ? x + 1.0 : std::exp(x)); }
inline double dphi(double x, int kind) { return kind == 1 ? (x > 0.0 ? 1.0 : 0.0) : (x > 0.0 ? 1.0 : std::exp(x)); }

// One window, one head, forward.  Rows s..e-1, head h.  Layout [N,H,d] row-major.
template <typename T>
void forward_window_head(const T* q, const T* k, const T* v, int64_t s, int64_t e, int H, int d, int h,
                         double* out, double* S /*d*d*/, double* z /*d*/, int kind, double eps) {
    for (int p = 0; p < d; ++p) { z[p] = 0.0; for (int r = 0; r < d; ++r) S[p * d + r] = 0.0; }
    for (int64_t j = s; j < e; ++j) {                       // S = sum_j phi(k_j)^T v_j ; z = sum_j phi(k_j)
        const T* kj = k + (j * H + h) * (int64_t)d;
        const T* vj = v + (j * H + h) * (int64_t)d;
        for (int p = 0; p < d; ++p) {
            double b = phi((double)kj[p], kind);
            z[p] += b;
            for (int r = 0; r < d; ++r) S[p * d + r] += b * (double)vj[r];
        }
    }
    std::vector<double> a(d);
    for (int64_t i = s; i < e; ++i) {                       // o_i = phi(q_i) S / (phi(q_i) . z + eps)
        const T* qi = q + (i * H + h) * (int64_t)d;
        double den = eps;
        for (int p = 0; p < d; ++p) { a[p] = phi((double)qi[p], kind); den += a[p] * z[p]; }
        double* oi = out + (i * H + h) * (int64_t)d;
        for (int r = 0; r < d; ++r) {
            double num = 0.0;
            for (int p = 0; p < d; ++p) num += a[p] * S[p * d + r];
            oi[r] = num / den;
        }
    }
}

// One window, one head, backward (derivatives of Eq. 3):
//   dnum_i = g_i/den_i ; dden_i = -(g_i.o_i)/den_i ; da_i = dnum_i S^T + dden_i z
//   dS = sum_i a_i^T dnum_i ; dz = sum_i dden_i a_i ; db_j = v_j dS^T + dz ; dv_j = b_j dS
//   dq_i = da_i * phi'(q_i) ; dk_j = db_j * phi'(k_j)
template <typename T>
void backward_window_head(const T* q, const T* k, const T* v, const T* g, int64_t s, int64_t e, int H,
                          int d, int h, double* dq, double* dk, double* dv, int kind, double eps) {
    std::vector<double> S(d * d), z(d), dS(d * d, 0.0), dz(d, 0.0), a(d), num(d), dnum(d);
    for (int p = 0; p < d; ++p) { z[p] = 0.0; for (int r = 0; r < d; ++r) S[p * d + r] = 0.0; }
    for (int64_t j = s; j < e; ++j) {
        const T* kj = k + (j * H + h) * (int64_t)d;
        const T* vj = v + (j * H + h) * (int64_t)d;
        for (int p = 0; p < d; ++p) {
            double b = phi((double)kj[p], kind);
            z[p] += b;
            for (int r = 0; r < d; ++r) S[p * d + r] += b * (double)vj[r];
        }
    }
    for (int64_t i = s; i < e; ++i) {
        const T* qi = q + (i * H + h) * (int64_t)d;
        const T* gi = g + (i * H + h) * (int64_t)d;
        double den = eps;                                   // "den" below is the whole denominator, eps included
        for (int p = 0; p < d; ++p) { a[p] = phi((double)qi[p], kind); den += a[p] * z[p]; }
        double go = 0.0;
        for (int r = 0; r < d; ++r) {
            double n = 0.0;
            for (int p = 0; p < d; ++p) n += a[p] * S[p * d + r];
            num[r] = n;
            double o = n / den;
            go += (double)gi[r] * o;
            dnum[r] = (double)gi[r] / den;
        }
        double dden = -go / den;
        double* dqi = dq + (i * H + h) * (int64_t)d;
        for (int p = 0; p < d; ++p) {
            double da = dden * z[p];
            for (int r = 0; r < d; ++r) da += dnum[r] * S[p * d + r];
            dqi[p] = da * dphi((double)qi[p], kind);
            dz[p] += dden * a[p];
            for (int r = 0; r < d; ++r) dS[p * d + r] += a[p] * dnum[r];
        }
    }
    for (int64_t j = s; j < e; ++j) {
        const T* kj = k + (j * H + h) * (int64_t)d;
        const T* vj = v + (j * H + h) * (int64_t)d;
        double* dkj = dk + (j * H + h) * (int64_t)d;
        double* dvj = dv + (j * H + h) * (int64_t)d;
        for (int r = 0; r < d; ++r) dvj[r] = 0.0;
        for (int p = 0; p < d; ++p) {
            double b = phi((double)kj[p], kind);
            double db = dz[p];
            for (int r = 0; r < d; ++r) { db += dS[p * d + r] * (double)vj[r]; dvj[r] += b * dS[p * d + r]; }
            dkj[p] = db * dphi((double)kj[p], kind);
        }
    }
}

// Static partition of windows over threads by voxel count (timed multi-thread variant only).
std::vector<int> partition_windows(const int32_t* off, int W, int nthreads) {
    std::vector<int> cuts(nthreads + 1, W);
    cuts[0] = 0;
    int64_t N = off[W];
    for (int t = 1; t < nthreads; ++t) {
        int64_t target = N * t / nthreads;
        cuts[t] = (int)(std::lower_bound(off, off + W + 1, (int32_t)target) - off);
        if (cuts[t] > W) cuts[t] = W;
        if (cuts[t] < cuts[t - 1]) cuts[t] = cuts[t - 1];
    }
    return cuts;
}

template <typename T>
void forward_impl(const T* q, const T* k, const T* v, const int32_t* off, int W, int H, int d,
                  double* out, double* S_out, double* z_out, int nthreads, int kind, double eps) {
    auto work = [&](int w0, int w1) {
        std::vector<double> S(d * d), z(d);
        for (int w = w0; w < w1; ++w) {
            int64_t s = off[w], e = off[w + 1];
            for (int h = 0; h < H; ++h) {
                double* Sp = S_out ? S_out + ((int64_t)w * H + h) * d * d : S.data();
                double* zp = z_out ? z_out + ((int64_t)w * H + h) * d : z.data();
                forward_window_head(q, k, v, s, e, H, d, h, out, Sp, zp, kind, eps);
            }
        }
    };
    if (nthreads <= 1) { work(0, W); return; }
    auto cuts = partition_windows(off, W, nthreads);
    std::vector<std::thread> th;
    for (int t = 0; t < nthreads; ++t) th.emplace_back(work, cuts[t], cuts[t + 1]);
    for (auto& x : th) x.join();
}

template <typename T>
void backward_impl(const T* q, const T* k, const T* v, const T* g, const int32_t* off, int W, int H,
                   int d, double* dq, double* dk, double* dv, int nthreads, int kind, double eps) {
    auto work = [&](int w0, int w1) {
        for (int w = w0; w < w1; ++w)
            for (int h = 0; h < H; ++h)
                backward_window_head(q, k, v, g, (int64_t)off[w], (int64_t)off[w + 1], H, d, h, dq, dk, dv, kind, eps);
    };
    if (nthreads <= 1) { work(0, W); return; }
    auto cuts = partition_windows(off, W, nthreads);
    std::vector<std::thread> th;
    for (int t = 0; t < nthreads; ++t) th.emplace_back(work, cuts[t], cuts[t + 1]);
    for (auto& x : th) x.join();
}

}  // namespace

extern "C" {

// Forward.  q,k,v: [N,H,d] row-major; off: int32[W+1]; out: double[N,H,d]; kind/eps: feature map (0 elu+1, 1 relu) and
// the epsilon added to the denominator;
// S_out (double[W,H,d,d]) and z_out (double[W,H,d]) may be NULL.
void sla_oracle_forward_f32(const float* q, const float* k, const float* v, const int32_t* off, int W,
                            int H, int d, double* out, double* S_out, double* z_out, int nthreads, int kind,
                            double eps) {
    forward_impl(q, k, v, off, W, H, d, out, S_out, z_out, nthreads, kind, eps);
}
void sla_oracle_forward_f64(const double* q, const double* k, const double* v, const int32_t* off, int W,
                            int H, int d, double* out, double* S_out, double* z_out, int nthreads, int kind,
                            double eps) {
    forward_impl(q, k, v, off, W, H, d, out, S_out, z_out, nthreads, kind, eps);
}

// Backward.  g = dL/dO, [N,H,d]; dq,dk,dv: double[N,H,d].
void sla_oracle_backward_f32(const float* q, const float* k, const float* v, const float* g,
                             const int32_t* off, int W, int H, int d, double* dq, double* dk, double* dv,
                             int nthreads, int kind, double eps) {
    backward_impl(q, k, v, g, off, W, H, d, dq, dk, dv, nthreads, kind, eps);
}
void sla_oracle_backward_f64(const double* q, const double* k, const double* v, const double* g,
                             const int32_t* off, int W, int H, int d, double* dq, double* dk, double* dv,
                             int nthreads, int kind, double eps) {
    backward_impl(q, k, v, g, off, W, H, d, dq, dk, dv, nthreads, kind, eps);
}

// Offsets prep (reading A10): off[w] = #{ i : win_id[i] < w }, w = 0..W,
// for non-decreasing ids in [0,W).  Written as the counting definition (O(N+W) via a histogram),
// tests pin it against std::lower_bound-style numpy.searchsorted and brute force.
void sla_oracle_offsets(const int32_t* win_id, int64_t N, int W, int32_t* off) {
    std::vector<int64_t> cnt(W + 1, 0);
    for (int64_t i = 0; i < N; ++i) cnt[win_id[i] + 1] += 1;   // cnt[w+1] = #{i : id == w}
    int64_t run = 0;
    for (int w = 0; w <= W; ++w) { run += cnt[w]; off[w] = (int32_t)run; }
}

int sla_oracle_hw_threads() { return (int)std::thread::hardware_concurrency(); }

}  // extern "C"
