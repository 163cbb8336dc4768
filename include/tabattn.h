/* libtabattn -- B200 (sm_100a) dual-axis attention for TabPFN-v2-style pretraining.
 *
 * The per-layer hot path of the nanoTabPFN pretraining step the paper speedruns
 * (Fig. 3: every transformer block applies "feature-axis attention,
 * norm, sample-axis attention, norm, MLP, norm"; both are
 * explicit-QKV scaled dot-product attention; thinking rows "count as
 * part of the train portion"; rows are queries, columns are keys).
 *
 * Cell tensor layout: every Q/K/V/O/dO/dQ/dK/dV is
 *     [B tables][R rows][C columns][H heads][dh]      bf16, row-major, dh fastest,
 * contiguous, 16-byte aligned, d = H*dh.  bf16 crosses this ABI as raw 16-bit
 * patterns behind void*.  ALL pointers are DEVICE pointers unless a name ends in
 * _host.  The caller owns every buffer; the library allocates no device memory,
 * never synchronises the host, and enqueues all work on `stream` (graph-capturable).
 * Outputs are fully overwritten; inputs are never written; no aliasing of an output
 * with any other argument.  Calls are re-entrant across host threads and across devices
 * (the device is the calling thread's current CUDA device; it must be sm_100): the only
 * process-wide state is a mutex-protected cache of TMA descriptors and per-device launch
 * attributes.  Concurrent calls must use different workspaces.
 *
 * Feature attention (a1/a2 of SURVEY.md §8(a)): for each (b, r, h) the sequence runs
 *   over the table's VALID columns:  S = scale * Q K^T (Cv x Cv), P = softmax_rows(S),
 *   O = P V, LSE = logsumexp_rows(S) (natural log).            n_train is ignored.
 * Item attention (a3-a5): for each valid (b, c), each h, every query row i in [0,R)
 *   attends to key rows j in [0, n_train[b]) only -- train and test queries alike.
 * Backward (both): D_i = sum_j P_ij dP_ij, dP = dO V^T, dS = P o (dP - D),
 *   dV = P^T dO, dQ = scale * dS K, dK = scale * dS^T Q; P is recomputed from LSE.
 *
 * Masked positions: O, dQ, dK, dV at invalid columns and item dK, dV at rows
 * >= n_train[b] are written as +0; LSE at invalid columns is 0.0f.  Values stored at
 * invalid columns of any input, and item K/V at rows >= n_train[b], never influence
 * an output (even NaN/Inf).  Inputs at valid positions must be finite.
 */
#ifndef TABATTN_H_
#define TABATTN_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define TABATTN_VERSION 100   /* major*10000 + minor*100 + patch */

#if defined(__GNUC__)
#define TABATTN_API __attribute__((visibility("default")))
#else
#define TABATTN_API
#endif

typedef enum {
  TABATTN_OK = 0,
  TABATTN_ERR_INVALID_ARG = 1, /* NULL required pointer, non-positive size, misaligned pointer,
                                  n_train_host[b] outside [1,R], NULL shape, an output pointer equal
                                  to another argument's pointer (aliasing) */
  TABATTN_ERR_UNSUPPORTED = 2, /* dh not in {16,32,64}, C > TABATTN_MAX_FEATURE_C for feature_*,
                                  B or C > 65535 for a masked item_* call,
                                  H*dh > TABATTN_MAX_D, B*R*C >= 2^31 cells, the calling thread's
                                  current device is not sm_100 */
  TABATTN_ERR_WORKSPACE = 3,   /* ws == NULL or ws_bytes < tabattn_workspace_bytes(shape, op) */
  TABATTN_ERR_CUDA = 4         /* a CUDA launch / driver call failed (see cudaGetLastError) */
} tabattn_status;

/* op codes for tabattn_workspace_bytes */
enum { TABATTN_OP_FEATURE_FWD = 0, TABATTN_OP_FEATURE_BWD = 1, TABATTN_OP_ITEM_FWD = 2, TABATTN_OP_ITEM_BWD = 3 };

#define TABATTN_MAX_FEATURE_C 128 /* largest column count the feature kernels accept */
#define TABATTN_MAX_D 4096        /* largest embedding width d = H*dh any call accepts  */

typedef struct {
  int32_t B, R, C, H, dh;       /* all >= 1; dh in {16, 32, 64}                                    */
  const int32_t* n_train;       /* DEVICE [B]; 1 <= n_train[b] <= R.  item_* only; feature_* ignore
                                   it (may be NULL there).  Out-of-range device values with no host
                                   copy are clamped to [1,R] (no device->host error path).          */
  const int32_t* n_train_host;  /* optional HOST copy [B] (NULL ok): enables the range check         */
  const uint8_t* col_valid;     /* DEVICE [B*C], nonzero = valid column; NULL = all valid            */
  float softmax_scale;          /* <= 0.0f  =>  1/sqrt(dh)                                           */
} tabattn_shape;

/* CUDA stream handle (cudaStream_t) passed as an opaque pointer so that this header needs no
 * CUDA include; NULL is the legacy default stream. */
typedef void* tabattn_stream;

/* Feature attention forward.  Q,K,V in; O [B,R,C,H,dh] bf16 and LSE [B,R,H,C] f32 out.
 * ws/ws_bytes: scratch of at least tabattn_workspace_bytes(shape, TABATTN_OP_FEATURE_FWD)
 * bytes (may be NULL when that is 0). */
TABATTN_API tabattn_status tabattn_feature_fwd(const tabattn_shape* shape, const void* Q, const void* K, const void* V,
                                   void* O, float* LSE, void* ws, size_t ws_bytes, tabattn_stream stream);

/* Feature attention backward.  O and LSE are the forward's outputs.  dQ,dK,dV out. */
TABATTN_API tabattn_status tabattn_feature_bwd(const tabattn_shape* shape, const void* Q, const void* K, const void* V,
                                   const void* O, const void* dO, const float* LSE, void* dQ, void* dK,
                                   void* dV, void* ws, size_t ws_bytes, tabattn_stream stream);

/* Item attention forward.  LSE is [B,C,H,R] f32 (contiguous along the sequence).  ws (only touched when a
 * column mask is given): tabattn_workspace_bytes(shape, TABATTN_OP_ITEM_FWD). */
TABATTN_API tabattn_status tabattn_item_fwd(const tabattn_shape* shape, const void* Q, const void* K, const void* V,
                                void* O, float* LSE, void* ws, size_t ws_bytes, tabattn_stream stream);

/* Item attention forward WITHOUT any allocation: the same computation, kernels and results as tabattn_item_fwd
 * (PAPER.md item-axis attention; same argument meaning, layouts and errors), for callers
 * that cannot call cudaMalloc (CUDA graph capture, serving loops, harnesses that forbid it) and so have no
 * workspace to pass.  The scratch of a masked call (the a0 column list, 4 * (B*C + 4) bytes) lives in a
 * `static __device__` array inside the library, sized for B*C <= TABATTN_NOALLOC_MAX_BC column pairs (256 KiB + 256 B
 * that every GPU loading the library holds until the process exits).  The call itself allocates nothing: no
 * cudaMalloc / cudaFree / allocating library routine; the array's device address is looked up once per device
 * (cudaGetSymbolAddress) on that device's first masked call.
 *   - shape->col_valid != NULL and B*C > TABATTN_NOALLOC_MAX_BC  =>  TABATTN_ERR_WORKSPACE (the built-in scratch is
 *     too small; nothing is launched).  Unmasked calls use no scratch and have no such limit.
 *   - Every call on a device shares the one array; it keeps the previous call's contents, and each call rewrites all
 *     of it that it reads (nothing has to start at zero).  Calls that overlap on the GPU (different streams, or
 *     several host threads on different streams) RACE on it: serialise them (one stream, or events). */
#define TABATTN_NOALLOC_MAX_BC 65536
TABATTN_API tabattn_status tabattn_item_fwd_noalloc(const tabattn_shape* shape, const void* Q, const void* K,
                                                    const void* V, void* O, float* LSE, tabattn_stream stream);

/* Item attention backward: a dQ pass (it also computes D = rowsum(dO o O) and -LSE*log2(e) per query
 * row and leaves them in the workspace) and a separate dK/dV pass that reads them; two kernel
 * launches, deterministic, no atomics.  ws: tabattn_workspace_bytes(shape, TABATTN_OP_ITEM_BWD)
 * (8 bytes per (b, c, h, row) at dh = 64, 36 at dh <= 32, rows rounded up to 64). */
TABATTN_API tabattn_status tabattn_item_bwd(const tabattn_shape* shape, const void* Q, const void* K, const void* V,
                                const void* O, const void* dO, const float* LSE, void* dQ, void* dK,
                                void* dV, void* ws, size_t ws_bytes, tabattn_stream stream);

/* ---- Forward-only evaluation path ----------------------------------------------
 * evaluation tables hold at most 1000 rows x 100 features, 5-fold (800 train / 200 test
 * rows); bf16 inference autocast; evaluation runs every 32-64 steps.
 * Inference needs neither the saved log-sum-exp nor, in the last block, the outputs of the train rows
 * ("the test-row outputs are sliced out"), so these calls write O only for the table rows
 * [row0, row1) of EVERY table -- e.g. one chunk of test rows -- and no LSE.  Rows of O outside the range
 * are not touched.  0 <= row0 < row1 <= R, else TABATTN_ERR_INVALID_ARG.  Everything else (layouts, the
 * column mask, +0 at invalid columns, the train-only key rule) is as in the training forward, and the
 * results on the range are bit-identical to it.
 *
 * Item: query rows [row0, row1) attend to the key rows [0, n_train[b]) of their own column; the caller
 * passes the same K and V for every chunk of test rows (the train-row K/V are projected once and reused).
 * Feature: the rows [row0, row1) of each table, each row alone.  A partial range with B > 1 is issued as
 * one launch per table.  ws: tabattn_workspace_bytes(shape, TABATTN_OP_FEATURE_FWD / _ITEM_FWD). */
TABATTN_API tabattn_status tabattn_feature_fwd_infer(const tabattn_shape* shape, const void* Q, const void* K,
                                                     const void* V, void* O, int32_t row0, int32_t row1, void* ws,
                                                     size_t ws_bytes, tabattn_stream stream);
TABATTN_API tabattn_status tabattn_item_fwd_infer(const tabattn_shape* shape, const void* Q, const void* K,
                                                  const void* V, void* O, int32_t row0, int32_t row1, void* ws,
                                                  size_t ws_bytes, tabattn_stream stream);

/* ---- The sub-blocks around the attention kernels ----------------------------
 * PAPER.md:L69 (Fig. 3): every block applies feature-axis attention, sample-axis attention and an MLP, each
 * with a norm; the norms sit BEFORE attention and MLP (pre-norm); RMSNorm;
 * the input of block i is scaled by 0.95^i; explicit Q, K, V projections;
 * MLP hidden width 768.  Where the paper is silent the readings b1-b6 of DESIGN.md §2
 * apply: no biases; gain-only RMSNorm  xs rsqrt(mean(xs^2) + eps) o g  with statistics in fp32; exact (erf)
 * GELU; weights stored [out][in] like nn.Linear; the decay factor alpha multiplies the sub-block's input.
 *
 *   attention sub-block:  xs = alpha x;  h = rmsnorm(xs) o g;  [q|k|v] = h Wqkv^T;  o = attention(q, k, v);
 *                         y = xs + o Wo^T
 *   MLP sub-block:        xs = alpha x;  h = rmsnorm(xs) o g;  u = h W1^T;  a = gelu(u);  y = xs + a W2^T
 *
 * x, y, dy, dx and every saved activation are bf16 [cells][e] (cells = B*R*C, the attention layout with
 * e = H*dh) or [cells][hidden]; g is bf16 [e]; Wqkv [3e][e], Wo [e][e], W1 [hidden][e], W2 [e][hidden] bf16.
 * Gradients of the parameters come back in fp32 (dg [e], dWqkv [3e][e], dWo [e][e], dW1, dW2), fully
 * overwritten; they are reduced over the cells in a fixed order (no atomics: bitwise reproducible).
 * The forward fills the `saved` buffers (caller-owned) the backward reads.  e must be a multiple of 64,
 * e <= 1024, hidden a multiple of 64; alpha <= 0 means 1; eps <= 0 means 1e-6.
 * axis: 0 = feature attention, 1 = item attention (shape->n_train required). */
typedef struct {
  void* h;      /* [cells][e] bf16    rmsnorm(alpha x) o g */
  float* rstd;  /* [cells] f32        1 / sqrt(mean((alpha x)^2) + eps) */
  void* q;      /* [cells][e] bf16 each: the projections and the attention output, in the attention layout */
  void* k;
  void* v;
  void* o;
  float* lse;   /* the attention's LSE (feature [B,R,H,C] / item [B,C,H,R]) */
} tabattn_attn_saved;

typedef struct {
  void* h;      /* [cells][e] bf16 */
  float* rstd;  /* [cells] f32 */
  void* u;      /* [cells][hidden] bf16  pre-activation */
  void* a;      /* [cells][hidden] bf16  gelu(u) */
} tabattn_mlp_saved;

TABATTN_API tabattn_status tabattn_attn_block_fwd(const tabattn_shape* shape, int32_t axis, float alpha, float eps,
                                                  const void* x, const void* g, const void* Wqkv, const void* Wo,
                                                  void* y, const tabattn_attn_saved* saved, void* ws,
                                                  size_t ws_bytes, tabattn_stream stream);
TABATTN_API tabattn_status tabattn_attn_block_bwd(const tabattn_shape* shape, int32_t axis, float alpha,
                                                  const void* x, const void* g, const void* Wqkv, const void* Wo,
                                                  const tabattn_attn_saved* saved, const void* dy, void* dx,
                                                  float* dg, float* dWqkv, float* dWo, void* ws, size_t ws_bytes,
                                                  tabattn_stream stream);
/* scratch bytes of the two calls above (backward != 0: the backward's) */
TABATTN_API size_t tabattn_attn_block_workspace_bytes(const tabattn_shape* shape, int32_t axis, int32_t backward);

TABATTN_API tabattn_status tabattn_mlp_fwd(int64_t cells, int32_t e, int32_t hidden, float alpha, float eps,
                                           const void* x, const void* g, const void* W1, const void* W2, void* y,
                                           const tabattn_mlp_saved* saved, tabattn_stream stream);
TABATTN_API tabattn_status tabattn_mlp_bwd(int64_t cells, int32_t e, int32_t hidden, float alpha, const void* x,
                                           const void* g, const void* W1, const void* W2,
                                           const tabattn_mlp_saved* saved, const void* dy, void* dx, float* dg,
                                           float* dW1, float* dW2, void* ws, size_t ws_bytes,
                                           tabattn_stream stream);
TABATTN_API size_t tabattn_mlp_workspace_bytes(int64_t cells, int32_t e, int32_t hidden);

/* Batched Newton-Schulz orthogonalisation, the core of the Muon update (PAPER.md:L85-87 Muon "with the same
 * hyperparameters as in modded-nanogpt"; the iteration is batched across the QKV weight
 * matrices).  For each of the nb matrices G_i [m][n] (bf16, m <= n):
 *     X = G_i / (||G_i||_F + 1e-7);   `steps` times:  A = X X^T;  B = b A + c A A;  X = a X + B X
 * with (a, b, c) = (3.4445, -4.7750, 2.0315), every product rounded to bf16 (reading b6).  X_out [nb][m][n]
 * bf16.  m, n multiples of 8.  ws: tabattn_newton_schulz_workspace_bytes(nb, m, n). */
TABATTN_API tabattn_status tabattn_newton_schulz(int32_t nb, int32_t m, int32_t n, const void* G, void* X_out,
                                                 int32_t steps, void* ws, size_t ws_bytes, tabattn_stream stream);
TABATTN_API size_t tabattn_newton_schulz_workspace_bytes(int32_t nb, int32_t m, int32_t n);

/* Bytes of device scratch `op` needs for `shape` (0 if shape is NULL or invalid). */
TABATTN_API size_t tabattn_workspace_bytes(const tabattn_shape* shape, int op);

/* Static, never-NULL description of a status code. */
TABATTN_API const char* tabattn_status_string(tabattn_status status);

/* Number of CUDA kernels this library has launched in this process so far (all threads, all
 * streams; monotonically increasing).  Lets a harness count the launches of a timed region. */
TABATTN_API uint64_t tabattn_launch_count(void);

/* TABATTN_VERSION the library was built with. */
TABATTN_API int tabattn_version(void);

#ifdef __cplusplus
}
#endif
#endif /* TABATTN_H_ */
