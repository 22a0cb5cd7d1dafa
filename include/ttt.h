/*
 * ttt.h — C ABI of the B200-native TTT global-context-memory hot path (Scal3R,
 * arxiv/paper_2604_08542). One context = the fast weights ("adaptive memory units") of nh
 * independent heads plus the workspaces the kernels need. Everything behind these calls runs in
 * hand-written CUDA kernels for sm_100a; there is no CPU fallback.
 *
 * The operations (PAPER.md = /root/reference/PAPER.md of the build; line numbers cited):
 *   network   f_W(x) = W2 ( SiLU(W1 x) o (W3 x) ), no bias                 Eq. 12
 *   update    W <- W - grad_W  sum_{i=1..M} eta_i L(f_W(k_i), v_i)          Eq. 8,
 *   loss      L(f_W(K), V) = sum_i - f_W(k_i)^T v_i                         Eq. 9,
 *   apply     o = f_W(q) with the UPDATED weights                           Eq. 4,
 *   chunks are processed one after another, W carried
 * Row-vector storage (reading P3): y = x W, W1,W3 in R^{hd x H}, W2 in R^{H x hd}.
 * The paper-silent options BASELINE.json requires (Newton-Schulz orthonormalised gradient,
 * fan-in re-normalisation) are defined in DESIGN.md, readings R-NS and R-RENORM.
 *
 * Conventions for every function below
 *   - returns TTT_OK (0) or a negative ttt_status; never throws, aborts, prints or reads the
 *     environment;
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream); all work is
 *     enqueued asynchronously on it; calls on one context must be stream-ordered by the caller;
 *   - every data pointer is a DEVICE pointer on cfg.device unless it says "host"; pointers are
 *     BORROWED for the call and must stay valid until the enqueued work has completed; every call
 *     makes cfg.device current for its own duration and restores the caller's device;
 *   - the context OWNS the fp32 master weights, their 16-bit operand copies, the partial-gradient
 *     and Newton-Schulz workspaces and the initial fan-in norms;
 *   - a context is not thread-safe; distinct contexts are independent.
 * Token tensors Q, K, V, O: [M][nh][hd] token-major, heads interleaved in the last dimension
 * (PAPER.md:376), element type cfg.act_dtype, row stride `ld` ELEMENTS (ld >= nh*hd).
 * Learning rates lr: [nh][M] fp32, one eta_i per head and token (reading P7).
 */
#ifndef TTT_B200_H
#define TTT_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ttt_ctx ttt_ctx;

typedef enum {
  TTT_OK = 0,
  TTT_ERR_ARG = -1,         /* NULL pointer / negative size / bad enum                         */
  TTT_ERR_SHAPE = -2,       /* M > max_tokens, ld < nh*hd, shape outside the supported set     */
  TTT_ERR_ALIGN = -3,       /* pointer not 16-byte aligned or ld*sizeof(elt) not a multiple of 16 */
  TTT_ERR_STATE = -4,       /* update/apply before ttt_init                                     */
  TTT_ERR_UNSUPPORTED = -5, /* combination the kernels do not implement (never a silent fallback) */
  TTT_ERR_NOMEM = -6,       /* cudaMalloc failed                                                */
  TTT_ERR_CUDA = -7         /* any other CUDA error; text in ttt_last_error                     */
} ttt_status;

typedef enum {
  TTT_F32 = 0,  /* Q,K,V,O fp32; every contraction in fp32 FFMA (parity config 1, tol 1e-4)   */
  TTT_BF16 = 1  /* Q,K,V,O bf16, fp32 master weights, tcgen05 MMAs with fp32 accumulation. Shapes the
                   tensor kernels take: hd = 64 with hidden <= 256; hd = 128 with any hidden
                   (<= 1024 with Newton-Schulz) — a hidden size that is not a multiple of 128 runs
                   zero-padded to the next one; hd a multiple of 256 up to 2048 with hidden a
                   multiple of 128 and ns_iters = renorm = 0 (the paper's own shape: nh = 1, hd = 1024,
                   hidden 1024..4096; three bf16 activation arrays of
                   max_tokens x nh x hidden are allocated). Any other shape with hd <= 128: ttt_create
                   returns TTT_ERR_UNSUPPORTED, unless cfg.cuda_core_fallback = 1 asks for the fp32
                   CUDA-core kernels behind a bf16 <-> fp32 conversion (hd % 8 == 0; same semantics,
                   ~40x slower); hd > 128 otherwise: TTT_ERR_SHAPE.
                   hd 64 / 128: token values are MMA operands as fp16 (converted on chip, exact for
                   magnitudes in [2^-14, 65504]; smaller ones keep an absolute error <= 2^-25, larger
                   ones clamp); hd >= 256: bf16 operands throughout. */
} ttt_dtype;

typedef struct {
  int32_t nh;                 /* heads (independent fast-weight sets, Eq. 13)    */
  int32_t hd;                 /* head dimension: f32 <= 128, multiple of 4; bf16 see ttt_dtype    */
  int32_t hidden;             /* H = hd*k, multiple of 4 (tensor paths: see ttt_dtype)           */
  int32_t act_dtype;          /* ttt_dtype of Q,K,V,O                                          */
  int32_t ns_iters;           /* 0 = plain gradient step (Eq. 8); n>0 = n Newton-Schulz iters  */
  int32_t renorm;             /* 0/1: restore each unit's fan-in 2-norm of ttt_init after update */
  int32_t linear_fast_weight; /* 0 = SwiGLU (Eq. 12); 1 = f_W(x) = x W1 closed-form test mode
                                 (needs hidden == hd; f32 path only)                           */
  int32_t device;             /* CUDA device ordinal                                           */
  int64_t max_tokens;         /* largest M of any later call (workspace sizing)                */
  int32_t cuda_core_fallback; /* TTT_BF16 only. 0: shapes without a tcgen05 kernel are rejected;
                                 1: they run on the fp32 CUDA-core kernels (explicit opt-in)      */
  int32_t reserved;           /* must be 0                                                     */
} ttt_config;

/* Create a context on cfg->device. `*out` is written only on success; on failure
 * ttt_create_error() describes why (thread-local static text, valid until the thread's next
 * ttt_create). */
int ttt_create(ttt_ctx** out, const ttt_config* cfg);
const char* ttt_create_error(void);

/* Which kernels the context's two call families run on: 1 = tcgen05 tensor-core kernels,
 * 0 = fp32 CUDA-core kernels (TTT_F32 contexts, or cfg.cuda_core_fallback). Either pointer may be NULL. */
int ttt_kernel_path(const ttt_ctx* ctx, int* update_on_tensor_cores, int* apply_on_tensor_cores);

/* Free everything the context owns. NULL is allowed. Synchronises the device. */
void ttt_destroy(ttt_ctx* ctx);

/* Load the initial fast weights (DEVICE, fp32, row-major): W1, W3 [nh][hd][H], W2 [nh][H][hd].
 * Records each unit's initial fan-in 2-norm (columns of W1/W3, length hd; columns of W2,
 * length H) for cfg.renorm, refreshes the 16-bit operand copies and drops any pending gradient.
 * May be called again at any time = reset of the memory (new sequence). */
int ttt_init(ttt_ctx* ctx, const float* W1, const float* W2, const float* W3, void* stream);

/* update (Eq. 8 with Eq. 9 and Eq. 12): gradient of sum_i lr[h][i] * (-f_W(k_i)^T v_i) over all
 * M tokens at the PRE-update weights, optional Newton-Schulz of each of the three gradient
 * matrices, W <- W - G, optional re-normalisation. K, V: [M][nh][hd] act_dtype, row stride ld.
 * lr: [nh][M] fp32. loss: optional DEVICE [nh] fp32 out = the differentiated quantity per head
 * (NULL = not computed). M == 0 is a no-op. */
int ttt_update(ttt_ctx* ctx, const void* K, const void* V, const float* lr, int64_t M,
               int64_t ld, float* loss, void* stream);

/* apply (Eq. 4): O = f_W(Q) with the current weights. O has Q's layout and dtype and must not
 * alias Q. M == 0 is a no-op. */
int ttt_apply(ttt_ctx* ctx, const void* Q, void* O, int64_t M, int64_t ld, void* stream);

/* chunk step: ttt_update(K,V,lr) then ttt_apply(Q) on the same stream, one launch
 * chain. Bitwise identical to the two calls made separately. */
int ttt_chunk_step(ttt_ctx* ctx, const void* Q, const void* K, const void* V, const float* lr,
                   void* O, int64_t M, int64_t ld, float* loss, void* stream);

/* Gradient accumulation without a weight change (Eq. 10: the gradient of a sum
 * of chunks at the same W is the sum of the chunks' gradients): adds this chunk's partial
 * gradients to the context's pending set. ttt_commit applies the pending set as ONE update
 * ([Newton-Schulz] -> W <- W - G -> [renorm]) and clears it. ttt_update == accumulate; commit.
 * A multi-GPU caller all-reduces ttt_pending_gradient() between the two (multi-GPU). */
int ttt_accumulate(ttt_ctx* ctx, const void* K, const void* V, const float* lr, int64_t M,
                   int64_t ld, float* loss, void* stream);
int ttt_commit(ttt_ctx* ctx, void* stream);

/* Reduce the pending partial gradients into one dense DEVICE buffer owned by the context and
 * return it: [3][nh][H'][hd] fp32 = (G1^T, G2, G3^T) in the hidden-major layout the kernels use
 * (H' = *n_elements / (3 nh hd): H, or — bf16 tensor path with hd 64 | 128 and H not a multiple of
 * 128 — H rounded up to one; the padded hidden units' rows are zero).
 * After the caller has modified it in place (e.g. ncclAllReduce), ttt_commit uses it as is. */
int ttt_pending_gradient(ttt_ctx* ctx, float** G, int64_t* n_elements, void* stream);

/* Copy the current fp32 fast weights out (DEVICE buffers in ttt_init's layout). */
int ttt_get_weights(ttt_ctx* ctx, float* W1, float* W2, float* W3, void* stream);

/* Number of kernels the context has launched since creation (bench accounting). */
int64_t ttt_launch_count(const ttt_ctx* ctx);

/* Static description of a status code / detail text of the last failure on this context. */
const char* ttt_strerror(int status);
const char* ttt_last_error(const ttt_ctx* ctx);

/* Library version string, e.g. "ttt-b200 0.1 (sm_100a)". */
const char* ttt_version(void);

#ifdef __cplusplus
}
#endif
#endif /* TTT_B200_H */
