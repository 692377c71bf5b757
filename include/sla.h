/* sla.h -- C ABI of the B200-native Scattered Linear Attention (SLA) library.
 *
 * Operation (ScatterFormer, arxiv 2401.00912; citations are PAPER.md line numbers):
 *   All voxels of a scene are one flat sequence ordered by window; window w owns rows
 *   off[w] .. off[w+1]-1.  SLA(Q,K,V) = Concat_w LA(Q^w,K^w,V^w)                 (Eq. 2)
 *   LA:  o_i = phi(q_i) S_w / (phi(q_i) . z_w),  S_w = sum_j phi(k_j)^T v_j  (d_h x d_h),
 *        z_w = sum_j phi(k_j)  (d_h),  sums over the voxels j of the window      (Eq. 3)
 *   applied independently per head.  phi(x) = elu(x)+1 = (x>0 ? x+1 : exp(x)), the map
 *   of the linear attention "[17]" that Eq. 3 cites; no epsilon, no 1/sqrt(d), non-causal
 *   (DESIGN.md "Readings" A1-A4).
 *
 * Conventions for every entry point
 *   - Pointers marked DEV are device pointers valid on the current CUDA device; HOST are host pointers.
 *   - Tensors q,k,v,out,d_out,dq,dk,dv are contiguous row-major [N, H, d_h] of `dt`
 *     (SLA_F32 / SLA_F16 / SLA_BF16); base pointers 16-byte aligned; H*d_h*sizeof(dt) a multiple of 16.
 *   - window_offsets: int32[W+1], off[0]=0, off[W]=N, non-decreasing (zero-length windows legal and
 *     produce nothing).  Violations are undefined behaviour (not checked on the device).
 *   - The caller owns every buffer, including `workspace`; the library never frees or keeps them.
 *     Inputs are read-only; outputs must not alias inputs.
 *   - Device entry points only enqueue work on `stream` and return; they never synchronise.
 *   - Return value: sla_status_t.  Never throws, never exits.  N==0 or W==0 -> SLA_OK, nothing launched.
 *   - d_h in {16, 32}.  1 <= H.  N < 2^31.
 *   - Accumulation is fp32 for every dtype; outputs are rounded (RNE) to `dt`.
 */
#ifndef SLA_H_
#define SLA_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  SLA_OK = 0,
  SLA_ERR_INVALID_ARG = 1,  /* NULL pointer, negative size, N >= 2^31 */
  SLA_ERR_UNSUPPORTED = 2,  /* d_h not in {16,32}, misaligned pointer, bad dtype */
  SLA_ERR_WORKSPACE = 3,    /* workspace NULL or smaller than sla_workspace_bytes() */
  SLA_ERR_CUDA = 4,         /* a CUDA runtime call failed (sticky error left for the caller) */
  SLA_ERR_TOO_LARGE = 5     /* sla_forward_static: the problem needs more than SLA_STATIC_WORKSPACE_BYTES of scratch */
} sla_status_t;

typedef enum { SLA_F32 = 0, SLA_F16 = 1, SLA_BF16 = 2 } sla_dtype_t;

/* Feature map phi of Eq. 3 ("phi(x) is the kernel function"; the paper never writes it out):
 *   SLA_PHI_ELU1  phi(x) = elu(x)+1, the map of the linear attention [17] that Eq. 3 cites; strictly
 *                 positive, so the denominator needs no epsilon.  What sla_forward / sla_backward compute.
 *   SLA_PHI_RELU  phi(x) = max(x, 0), the "Efficient Attn [3]" kernel that labels Table 7's default row
 *                 (PAPER.md:277, 296), with an epsilon added to the denominator (which can otherwise be exactly 0):
 *                 o_i = phi(q_i) S / (phi(q_i) . z + eps).  Entry points sla_forward_phi / sla_backward_phi. */
typedef enum { SLA_PHI_ELU1 = 0, SLA_PHI_RELU = 1 } sla_feature_map_t;

/* Opaque CUDA stream handle (a cudaStream_t / CUstream); NULL = the legacy default stream. */
typedef struct CUstream_st* sla_stream_t;

/* Human-readable name of a status code (static storage). */
const char* sla_status_string(int status);

/* Library version string, e.g. "sla-b200 0.1 (sm_100a)". */
const char* sla_version(void);

/* Bytes of device workspace sla_forward (for_backward=0) or sla_backward (for_backward=1) needs for a
 * problem of this shape.  The workspace holds the fp32 window states [W,H,d_h+1,d_h] of windows that
 * are split across thread blocks (row d_h of each state is z_w), and for backward also dS/dz.
 * Returns 0 on invalid arguments. */
size_t sla_workspace_bytes(int64_t N, int32_t W, int32_t H, int32_t d_h, int dt, int for_backward);

/* Offsets prep ("offsets generation", Fig. 5; flat window-sorted layout PAPER.md:77).
 *   win_id          DEV int32[N]   window index of each voxel, non-decreasing, each in [0, W); a tail of ids
 *                                  equal to W ("no window", see sla_window_keys) is accepted
 *   window_offsets  DEV int32[W+1] out: off[w] = #{ i : win_id[i] < w }   (bit-exact integer result)
 * Gaps in the ids give zero-length windows (reading A10). */
int sla_offsets_from_window_ids(const int32_t* win_id, int64_t N, int32_t W,
                                int32_t* window_offsets, sla_stream_t stream);

/* SLA forward (Eq. 2-3).
 *   q,k,v           DEV [N,H,d_h] of dt (read-only)
 *   window_offsets  DEV int32[W+1]
 *   out             DEV [N,H,d_h] of dt
 *   workspace       DEV, >= sla_workspace_bytes(N,W,H,d_h,dt,0) bytes, 16-byte aligned; contents
 *                   are scratch (overwritten). */
int sla_forward(const void* q, const void* k, const void* v, const int32_t* window_offsets,
                int64_t N, int32_t W, int32_t H, int32_t d_h, int dt, void* out,
                void* workspace, size_t workspace_bytes, sla_stream_t stream);

/* sla_forward / sla_backward with the feature map chosen by the caller (sla_feature_map_t) and `eps` added to the
 * denominator of Eq. 3 (eps >= 0; must be 0 for SLA_PHI_ELU1, > 0 recommended for SLA_PHI_RELU, e.g. 1e-6).  All other
 * arguments, the workspace size and the error behaviour are those of sla_forward / sla_backward, which are these
 * calls with (SLA_PHI_ELU1, 0).  Unknown map or eps < 0 -> SLA_ERR_INVALID_ARG.  Backward of the ReLU map:
 * phi'(x) = 1 for x > 0, else 0. */
int sla_forward_phi(const void* q, const void* k, const void* v, const int32_t* window_offsets,
                    int64_t N, int32_t W, int32_t H, int32_t d_h, int dt, int feature_map, float eps, void* out,
                    void* workspace, size_t workspace_bytes, sla_stream_t stream);
int sla_backward_phi(const void* q, const void* k, const void* v, const int32_t* window_offsets,
                     int64_t N, int32_t W, int32_t H, int32_t d_h, int dt, int feature_map, float eps,
                     const void* d_out, void* dq, void* dk, void* dv,
                     void* workspace, size_t workspace_bytes, sla_stream_t stream);

/* The same operation as sla_forward, same arguments and results within the same tolerance, with the main pass on
 * the 5th-generation tensor cores (tcgen05.mma, accumulators in tensor memory; csrc/sla_fwd_umma.cu): all heads of a
 * 128-channel slab in one MMA per 16 rows.  Supported: dt = SLA_F16, d_h = 16, H*d_h a multiple of 128; anything
 * else -> SLA_ERR_UNSUPPORTED.  It is parity-tested like sla_forward but slower on the measured scenes (DESIGN.md
 * 5.7), so sla_forward does not route to it. */
int sla_forward_tcgen05(const void* q, const void* k, const void* v, const int32_t* window_offsets,
                        int64_t N, int32_t W, int32_t H, int32_t d_h, int dt, void* out,
                        void* workspace, size_t workspace_bytes, sla_stream_t stream);

/* sla_forward for callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc): the same operation, arguments, kernels and results as sla_forward, but the workspace is a
 * static device array inside the library, so the caller passes none and the call allocates nothing -- no cudaMalloc,
 * cudaFree or allocating library routine, in the library or asked of the caller.
 *   - The array has SLA_STATIC_WORKSPACE_BYTES (4 MiB); every GPU that loads the library holds it until exit.
 *   - A problem fits iff sla_workspace_bytes(N, W, H, d_h, dt, 0) <= SLA_STATIC_WORKSPACE_BYTES, i.e. about
 *     N * H * (d_h + 1) * d_h * 4 / 257 bytes: N up to ~123 000 voxels at H = 8, d_h = 16 (configs 1 and 4 fit, config 2
 *     does not).  Anything larger -> SLA_ERR_TOO_LARGE, nothing launched; call sla_forward with your own workspace.
 *   - All calls on one device share the array, and it keeps the previous call's contents: each call zeroes the part
 *     it uses on `stream` before its kernels run.  Calls that may overlap on the GPU (different streams, or graphs
 *     replayed concurrently) RACE on it; serialise them, or use sla_forward with one workspace per stream.
 *   - The array's device address is looked up once per device (cudaGetSymbolAddress) on the first call there. */
#define SLA_STATIC_WORKSPACE_BYTES (4u << 20)
int sla_forward_static(const void* q, const void* k, const void* v, const int32_t* window_offsets,
                       int64_t N, int32_t W, int32_t H, int32_t d_h, int dt, void* out, sla_stream_t stream);

/* SLA forward when the caller knows an upper bound on the window length.  In ScatterFormer a window
 * is a fixed block of BEV cells (12x12 on Waymo), so no window can hold more than 144
 * voxels: that bound is a model constant.  With 1 <= max_window_len <= 256 every window is processed
 * whole by one thread block, so the call is ONE kernel launch and needs no workspace.
 *   max_window_len  every window must satisfy off[w+1]-off[w] <= max_window_len (not checked on the
 *                   device; a longer window is undefined behaviour).  > 256 -> SLA_ERR_UNSUPPORTED
 *                   (call sla_forward instead).
 * Results are identical to sla_forward on the same inputs. */
int sla_forward_bounded(const void* q, const void* k, const void* v, const int32_t* window_offsets,
                        int64_t N, int32_t W, int32_t H, int32_t d_h, int dt, void* out,
                        int32_t max_window_len, sla_stream_t stream);

/* The work list of the flat sequence, built once per scene ("chunk -> window map / work list",
 * PAPER.md:93 Fig. 3a; the paper's "offsets generation" stage, Fig. 5): for every row span the tensor-core forward
 * hands to a thread block, the window of its first row and the rows the block streams.  A scene's window structure is
 * the same for every block of the network and for every head, so the table is built once and passed to every
 * sla_forward_planned call on that scene; without it every thread block finds its windows by a search of the offsets
 * (three dependent rounds of probes), with it by one 16-byte load.
 *   table  DEV, >= sla_span_table_bytes(N, H, d_h) bytes, 16-byte aligned; written by sla_build_span_table (one small
 *          kernel on `stream`), read-only afterwards; valid for this (window_offsets, N, H, d_h) on this device.
 *          Layout (int32, checked bit for bit by tests/test_gpu_parity.py against a CPU restatement): entry 0 =
 *          {magic, span, nspans, N}; entry 1 + i for the span of rows [i*span, min((i+1)*span, N)) =
 *          {w0, begin, end, 0}: w0 = the window that holds the span's first row; a window of <= 256 rows belongs to
 *          the span that holds its middle row off[w] + len/2, so begin = off[w0] if that middle is >= the span's first
 *          row, else off[w0+1]; end = off[wl+1] if the middle of wl (the window of the span's last row) lies inside the
 *          span, else off[wl]; longer windows are cut at the span's own borders (begin = first row, end = last row + 1).
 *          The rows streamed are [begin, max(begin, end)).
 * sla_forward_planned = sla_forward_bounded (same promise about max_window_len, same results bit for bit, one launch, no
 * workspace) + the table.  A table that belongs to another N or launch geometry is detected on the device and ignored
 * (the kernel searches as usual); a table of other offsets with the same N is undefined behaviour. */
size_t sla_span_table_bytes(int64_t N, int32_t H, int32_t d_h);
int sla_build_span_table(const int32_t* window_offsets, int64_t N, int32_t W, int32_t H, int32_t d_h,
                         void* table, size_t table_bytes, sla_stream_t stream);
int sla_forward_planned(const void* q, const void* k, const void* v, const int32_t* window_offsets,
                        int64_t N, int32_t W, int32_t H, int32_t d_h, int dt, void* out,
                        int32_t max_window_len, const void* table, size_t table_bytes, sla_stream_t stream);

/* SLA backward: gradients of L = sum(d_out * SLA(q,k,v)) (the paper is silent on backward; these are
 * the analytic derivatives of Eq. 3):
 *   dnum_i = g_i/den_i, dden_i = -(g_i.o_i)/den_i, da_i = dnum_i S^T + dden_i z, dq_i = da_i*phi'(q_i)
 *   dS = sum_i a_i^T dnum_i, dz = sum_i dden_i a_i, dk_j = (v_j dS^T + dz)*phi'(k_j), dv_j = b_j dS.
 *   d_out           DEV [N,H,d_h] of dt (upstream gradient g)
 *   dq,dk,dv        DEV [N,H,d_h] of dt (outputs)
 *   workspace       DEV, >= sla_workspace_bytes(N,W,H,d_h,dt,1) bytes.
 * The window states are recomputed from k,v; nothing is carried over from sla_forward. */
int sla_backward(const void* q, const void* k, const void* v, const int32_t* window_offsets,
                 int64_t N, int32_t W, int32_t H, int32_t d_h, int dt, const void* d_out,
                 void* dq, void* dk, void* dv,
                 void* workspace, size_t workspace_bytes, sla_stream_t stream);

/* sla_backward when the caller knows an upper bound on the window length (see sla_forward_bounded): with
 * 1 <= max_window_len <= 256 every window is differentiated whole by one thread block, so the call is ONE kernel
 * launch and needs no workspace.  A window longer than the promise is undefined behaviour (not checked on the device);
 * max_window_len > 256 -> SLA_ERR_UNSUPPORTED (call sla_backward).  Results are identical to sla_backward. */
int sla_backward_bounded(const void* q, const void* k, const void* v, const int32_t* window_offsets,
                         int64_t N, int32_t W, int32_t H, int32_t d_h, int dt,
                         const void* d_out, void* dq, void* dk, void* dv,
                         int32_t max_window_len, sla_stream_t stream);

/* End-to-end host entry (what a user with host data calls): copies q,k,v (and win_id) from HOST
 * memory to the device, runs sla_offsets_from_window_ids + sla_forward, copies `out` back to HOST
 * memory and synchronises `stream` before returning.  Device scratch is taken from a stream-ordered
 * CUDA memory pool that the library creates per device on first use (unbounded release threshold, so
 * the block is reused by the next call instead of going back to the driver) and is returned to that
 * pool before the call ends.  The scene is cut at window boundaries into up to four chunks; chunk c+1 is copied in while
 * chunk c is computed and chunk c-1 is copied out, on two copy streams the library creates per device on first use
 * (ordered against `stream` with events).  This is the only entry that owns device memory and streams; they live until
 * exit.  win_id must be non-decreasing with every id in [0, W) (checked at the chunk boundaries only).
 *   q,k,v   HOST [N,H,d_h] of dt (pinned memory recommended)      win_id  HOST int32[N]
 *   out     HOST [N,H,d_h] of dt */
int sla_forward_host(const void* q, const void* k, const void* v, const int32_t* win_id,
                     int64_t N, int32_t W, int32_t H, int32_t d_h, int dt, void* out,
                     sla_stream_t stream);

/* ---- Sequence preparation ------------------------------------------------------------------
 * "we arrange the voxels of the entire scene into a single flattened matrix ... ordered based on their window
 * coordinates, ensuring that voxels from the same window form a sub-matrix in contiguous memory";
 * windows are S_h x S_w cells of the ground plane.  Integer and byte work: every result below is
 * unique and bit-exact.  What the paper leaves open is fixed by DESIGN.md reading A16:
 *   - coords is int32[N,4], one row (b, z, y, x) per voxel: sample in the batch, then the cell, slowest axis first;
 *     z takes no part.  The key of a voxel is the row-major index of (b, y / S_h, x / S_w) among the
 *     W = batch * ceil(grid_h / S_h) * ceil(grid_w / S_w) windows; a voxel with b, y or x outside
 *     [0,batch) x [0,grid_h) x [0,grid_w) gets the key W ("no window"; it sorts behind every window).
 *   - The window-sorted order is the STABLE sort by key (voxels of one window keep their input order);
 *     perm[j] is the input position of the voxel at sorted position j.
 * All pointers DEV; every entry only enqueues kernels on `stream`.  N < 2^31, W < 2^31 - 1. */

/* W for this grid and window shape; -1 if an argument is < 1 or W does not fit. */
int64_t sla_window_count(int32_t batch, int32_t grid_h, int32_t grid_w, int32_t S_h, int32_t S_w);

/*   coords  DEV int32[N,4], 16-byte aligned (read-only)        key  DEV int32[N] out, each in [0, W] */
int sla_window_keys(const int32_t* coords, int64_t N, int32_t batch, int32_t grid_h, int32_t grid_w,
                    int32_t S_h, int32_t S_w, int32_t* key, sla_stream_t stream);

/* Bytes of device workspace sla_sort_by_window needs for N keys (0 on invalid N). */
size_t sla_sort_workspace_bytes(int64_t N);

/* Stable sort of the voxels by key (least-significant-digit radix sort, 8 bits per pass over the bits of W).
 *   key         DEV int32[N], each in [0, W] (read-only; a key outside that range is undefined behaviour)
 *   perm        DEV int32[N] out: a permutation of 0..N-1, key[perm[j]] non-decreasing in j, ties in input order
 *   key_sorted  DEV int32[N] out: key[perm[j]]; must not be `key`.  Feed it to sla_offsets_from_window_ids
 *               (which accepts the trailing keys equal to W: off[W] is then the number of voxels inside the grid).
 *   workspace   DEV, >= sla_sort_workspace_bytes(N) bytes, 16-byte aligned, scratch */
int sla_sort_by_window(const int32_t* key, int64_t N, int32_t W, int32_t* perm, int32_t* key_sorted,
                       void* workspace, size_t workspace_bytes, sla_stream_t stream);

/* dst[j] = src[perm[j]] for j in [0,N): input-order rows -> the window-sorted matrix.  Rows are `row_bytes` bytes,
 * a multiple of 4 (copied 16 bytes at a time when rows and both base pointers allow); src and dst 4-byte aligned and
 * distinct.  A row whose perm entry lies outside [0,N) is skipped (never read or written out of bounds). */
int sla_gather_rows(const void* src, const int32_t* perm, int64_t N, size_t row_bytes, void* dst, sla_stream_t stream);

/* dst[perm[j]] = src[j]: window-sorted rows (the op's output) back to input order; undoes sla_gather_rows. */
int sla_scatter_rows(const void* src, const int32_t* perm, int64_t N, size_t row_bytes, void* dst, sla_stream_t stream);

/* The three steps in one call: keys -> stable sort -> offsets.
 *   perm, key_sorted  DEV int32[N] out (as above)        window_offsets  DEV int32[W+1] out, W = sla_window_count(...)
 *   workspace         DEV, >= sla_sequence_workspace_bytes(N) bytes, 16-byte aligned, scratch
 * off[W] is the number of voxels inside the grid: pass that as N to sla_forward when some voxels lie outside.
 * With W + 1 <= 2048 (a single frame) the call is a counting sort in one pass -- two kernels, the offsets fall out of its
 * scan -- instead of keys + radix passes + offsets; same results bit for bit. */
size_t sla_sequence_workspace_bytes(int64_t N);
int sla_sequence_from_coords(const int32_t* coords, int64_t N, int32_t batch, int32_t grid_h, int32_t grid_w,
                             int32_t S_h, int32_t S_w, int32_t* perm, int32_t* key_sorted, int32_t* window_offsets,
                             void* workspace, size_t workspace_bytes, sla_stream_t stream);

/* ---- The shared Q/K/V projection around the op ------------------------------------------------
 * "Self-attention first linearly projects the input to queries, keys, and values ... Q = x W_Q, K = x W_K, V = x W_V"
 * (PAPER.md:71); "we use a shared projection layer to map all the voxels in the scene to query, key, and value
 * representations".  One GEMM y[N, 3C] = x[N, C] . w_qkv[3C, C]^T (+ bias) on the tensor cores
 * (tcgen05.mma, fp32 accumulation, one rounding to `dt`), written to three tensors (reading A17):
 *   x      DEV [N, C] of dt, C = H * d_h (read-only)
 *   w_qkv  DEV [3C, C] of dt: row j holds the weights of output feature j (the layout of a linear layer's weight);
 *          rows 0..C-1 give Q (W_Q of the paper is their transpose), C..2C-1 give K, 2C..3C-1 give V (read-only)
 *   bias   DEV fp32 [3C], 16-byte aligned, added before the rounding; NULL = none (the paper's formula has none)
 *   q,k,v  DEV [N, C] of dt out; as [N, H, d_h] they are what sla_forward takes
 * fp16 / bf16 with C in {128, 256} run on the tensor cores; fp32 I/O and every other C take a plain tiled kernel on the
 * CUDA cores (fp32 accumulation as well; a fallback, not a fast path).  All base pointers 16-byte aligned.  Enqueues one
 * kernel on `stream`; no workspace. */
int sla_qkv_projection(const void* x, const void* w_qkv, const float* bias, int64_t N, int32_t C, int dt,
                       void* q, void* k, void* v, sla_stream_t stream);

/* One linear layer with the same kernel: y[N, C] = x[N, C] . w[C, C]^T (+ bias), e.g. the output projection that follows
 * the attention in a transformer block (the paper's module implies one; it prints no formula for it).  w is [C, C], row j =
 * weights of output feature j; bias fp32 [C] or NULL; same support and alignment rules as sla_qkv_projection; x != y. */
int sla_linear(const void* x, const void* w, const float* bias, int64_t N, int32_t C, int dt, void* y,
               sla_stream_t stream);

/* The module of PAPER.md:77: projection, then SLA(Q, K, V) (Eq. 2-3): sla_qkv_projection followed by sla_forward on
 * the same stream (one chain of programmatic dependent launches; q, k, v stay in L2 between the two when 3 N C
 * elements fit there).  q, k, v are caller-owned outputs as well (a training step needs them for sla_backward);
 * workspace as for sla_forward.  Errors: those of the two calls. */
int sla_module_forward(const void* x, const void* w_qkv, const float* bias, const int32_t* window_offsets,
                       int64_t N, int32_t W, int32_t H, int32_t d_h, int dt,
                       void* q, void* k, void* v, void* out,
                       void* workspace, size_t workspace_bytes, sla_stream_t stream);

/* ---- Cross-Window Interaction (Eq. 4-7) --------------------------------------
 * "the input features are divided along the channel dimension and processed through multiple branches using
 * group-wise convolutions ... a (S_h+1) x 1 x 1 convolution in one branch and a 1 x (S_w+1) x 1 convolution in another
 * ... a standard 3 x 3 x 3 convolution in one branch ... while another branch performs an identity mapping":
 *   X' = Concat(DWConv_{S_h+1 along y}(X[:, 0:c]), DWConv_{S_w+1 along x}(X[:, c:2c]), DWConv_{3x3x3}(X[:, 2c:3c]), X[:, 3c:4c])
 * with C = 4c and depth-wise (per-channel) kernels.  DESIGN.md reading A18 fixes what the paper leaves open:
 *   - voxels are sparse: coords is int32[N,4], rows (b, z, y, x), all DISTINCT and inside
 *     [0,batch) x [0,grid_z) x [0,grid_h) x [0,grid_w); outputs live on the same voxels (row i of out <-> row i of x);
 *     a tap that lands on a cell without a voxel, outside the grid or in another sample contributes nothing.
 *     A voxel outside the grid is seen by nobody and gets zeros in the three convolution branches; duplicated
 *     coordinates give an unspecified one of the duplicates to their neighbours.  Nothing is read or written out of
 *     bounds either way.
 *   - S_h, S_w even (the window size): kernels of S+1 taps, centred, offsets -S/2..+S/2; 3x3x3 tap index
 *     (dz+1)*9 + (dy+1)*3 + (dx+1); cross-correlation: out[i] = sum_t w[t] * x[voxel at coords[i] + offset(t)].
 *   x, out   DEV [N, C] of dt (fp32 / fp16 / bf16), distinct buffers        coords  DEV int32[N,4], 16-byte aligned
 *   w_h      DEV fp32 [c, S_h+1]     w_w  DEV fp32 [c, S_w+1]     w_3  DEV fp32 [c, 27]     (no bias)
 *   workspace DEV, >= sla_cwi_workspace_bytes(batch, grid_z, grid_h, grid_w) = 4 bytes per grid cell (the dense
 *            voxel-index grid) + 4 bytes per (b, y, x) column (occupancy words), 16-byte aligned, scratch: its
 *            contents at entry do not matter and mean nothing afterwards
 * fp32 accumulation in tap order (deterministic), one rounding to dt.  C % 4 == 0, C <= 512, S_h + S_w <= 99, fewer
 * than 2^31 grid cells; otherwise SLA_ERR_UNSUPPORTED / SLA_ERR_INVALID_ARG.  Enqueues three kernels on `stream`. */
size_t sla_cwi_workspace_bytes(int32_t batch, int32_t grid_z, int32_t grid_h, int32_t grid_w);
int sla_cwi_forward(const void* x, const int32_t* coords, int64_t N, int32_t C, int dt,
                    int32_t batch, int32_t grid_z, int32_t grid_h, int32_t grid_w, int32_t S_h, int32_t S_w,
                    const float* w_h, const float* w_w, const float* w_3, void* out,
                    void* workspace, size_t workspace_bytes, sla_stream_t stream);

/* Measurement aid, not a step of the SLA path ("a size-matched pure read+write kernel
 * run beside config 1 as the practical ceiling").  Streams three tensors in and one out with 128-bit
 * accesses -- the forward's 3:1 read:write mix -- and nothing else: out = a ^ b ^ c, bytewise.
 *   a,b,c  DEV, `bytes` bytes each, 16-byte aligned (read-only)      out  DEV, `bytes` bytes
 *   bytes  a multiple of 16.  Enqueues one kernel on `stream`; never synchronises. */
int sla_bench_stream_ceiling(const void* a, const void* b, const void* c, void* out, size_t bytes,
                             sla_stream_t stream);

#ifdef __cplusplus
}
#endif
#endif /* SLA_H_ */
