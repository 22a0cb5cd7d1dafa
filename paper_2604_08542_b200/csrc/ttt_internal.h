// ttt_internal.h — context layout and launcher prototypes shared by the translation units of
// libttt_b200.so. Not part of the public ABI (that is include/ttt.h).
#pragma once

#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/ttt.h"

// Operand precision. Everything the library itself rounds to 16 bits
// for an MMA — the operand copy of the fp32 fast weights and the epilogue's gradient operands — is
// rounded to IEEE fp16 (11-bit significand, 8x finer than bf16). A kind::f16 MMA needs A and B in the
// SAME format (fp16 x bf16 raises an illegal-instruction fault on sm_100a — measured), so the bf16
// token tiles are converted to fp16 on chip before they serve as operands: exact for magnitudes in
// [2^-14, 65504], absolute error <= 2^-25 below. Saturating conversions: a value beyond +-65504
// clamps instead of turning into inf.
typedef __half ttt_wop_t;
constexpr int TTT_FMT_F16 = 0, TTT_FMT_BF16 = 1;     // instruction-descriptor format codes, kind::f16
constexpr int TTT_FMT_WOP = TTT_FMT_F16;
#ifdef __CUDACC__
__device__ __forceinline__ uint32_t ttt_pack_wop2(float lo, float hi) {   // `lo` in bits [0,16)
  uint32_t r;
  asm("cvt.rn.satfinite.f16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
  return r;
}
__device__ __forceinline__ ttt_wop_t ttt_to_wop(float v) {
  const uint32_t r = ttt_pack_wop2(v, 0.f);
  return __ushort_as_half(static_cast<unsigned short>(r & 0xffffu));
}
#endif

// Internal weight layout ("hidden-major"): three matrices per head, each [H][hd], hd contiguous:
//   mat 0 = W1^T   (row j = fan-in vector of hidden unit j of the gate branch, Eq. 12)
//   mat 1 = W2     (row j = fan-out vector of hidden unit j;  column o = fan-in of output o)
//   mat 2 = W3^T   (row j = fan-in vector of hidden unit j of the up branch)
// Element (mat, h, j, i) lives at ((mat*nh + h)*H + j)*hd + i, in the fp32 master `Wm`, the bf16
// operand copy `Wb`, the dense gradient `G` and every partial-gradient set.
struct ttt_ctx {
  ttt_config cfg;        // as the kernels see it: cfg.hidden is the PADDED hidden size (below)
  int user_hidden;       // the caller's H. bf16 tensor path with hd 64 | 128: H is padded to a multiple of 128
                         // with zero weight rows (zero units: x = b = g = 0, so their gradients and outputs
                         // vanish and the rows stay zero); ttt_init / ttt_get_weights translate
  int sm_count;
  bool initialised;
  int64_t launches;
  char err[512];

  size_t mat_elems;      // nh*H*hd
  float* Wm;             // [3][nh][H][hd] fp32 master weights
  ttt_wop_t* Wb;         // [3][nh][H][hd] 16-bit operand copy (fp16; refreshed by init/commit)
  __nv_bfloat16* Wq;     // hd = 128 only: bf16 copy for the apply kernel, whose Q tiles are SS-mode A
                         // operands straight from the TMA (bf16 x bf16 products); NULL otherwise
  float* n0;             // initial fan-in norms: [nh][H] (mat 0), [nh][hd] (mat 1), [nh][H] (mat 2)
  float* colsq;          // [nh][rowblocks][hd] partial column sums of squares of W2 (renorm)

  // pending gradient = (G_valid ? G : 0) + sum_{s < n_partials} partials[s], summed in this order
  float* G;              // [3][nh][H][hd]
  bool G_valid;
  float* partials;       // [cap_partials][3][nh][H][hd]
  int cap_partials;
  int n_partials;
  float* loss_part;      // [cap_loss_rows][nh] per-CTA-group loss partials of the last accumulate
  int cap_loss_rows;
  float* loss_blk;       // f32 path: per-block loss partials [nh][ceil(max_tokens/64)][ceil(H/64)]

  // f32 path workspaces: three [nh][max_tokens][H] fp32 activation buffers
  float* act[3];
  // bf16 I/O on the fp32 CUDA-core path (shapes the tensor kernels do not cover yet, e.g. hd = 128):
  // two [max_tokens][nh*hd] fp32 staging buffers for the converted token tensors
  bool upd_via_f32, app_via_f32;   // per call family: update (accumulate) / apply
  float* stage[2];

  // large-dimension path (hd >= 256, bf16_large.cu): hidden activations dA | dB | Hd' (update) and Hq
  // (apply, lact[0]) as bf16 [max_tokens][nh * hidden]; the pending gradient is the dense G only
  bool large;
  __nv_bfloat16* lact[3];

  // bf16 path: group-barrier counters of the fused commit ([nh][hidden/128]) and their running target
  // hd = 128 Newton-Schulz: partial Gram matrices [3 nh][hidden/128][2][128 x 128] fp32
  float* ns_scratch;
  unsigned* sync_ctr;
  unsigned sync_target;
  // set by ttt_chunk_step around its apply launch: Q may be requested before the PDL wait
  int apply_q_early;

  // bf16 path: driver entry point for cuTensorMapEncodeTiled
  void* encode_tiled;

  // per-context launch state (function attributes are per device; nothing process-global)
  uint32_t attr_done;          // bit k: the opt-in shared-memory size of kernel k has been set (ATTR_*)
  size_t attr_smem_apply, attr_smem_ns;   // high-water marks of the kernels with a shape-dependent size
  int max_pairs;               // hd = 128 apply: co-resident CTA pairs (0 = not queried yet, < 0 = none)
  int upd_coop_ctas;           // hd = 64 update: co-resident CTAs of the cooperative launch (0 = not queried)
  int ld_pairs;                // large-dimension path: co-resident CTA pairs of the forward kernel (0 = use single CTAs)
};
enum { ATTR_UPD = 1, ATTR_UPD_LOSS = 2, ATTR_UPDW = 4, ATTR_APPW = 8, ATTR_NSW = 16, ATTR_NS_F32 = 32,
       ATTR_LARGE = 64 };

namespace ttt {

int set_error(ttt_ctx* ctx, int status, const char* what, cudaError_t e);

// --- state kernels (state_kernels.cu) -----------------------------------------------------------
int launch_init(ttt_ctx* ctx, const float* W1, const float* W2, const float* W3, cudaStream_t s);
int launch_get_weights(ttt_ctx* ctx, float* W1, float* W2, float* W3, cudaStream_t s);
// G = (G_valid ? G : 0) + sum partials; marks G_valid, clears n_partials
int launch_reduce_pending(ttt_ctx* ctx, cudaStream_t s);
// [NS] -> W -= pending -> [renorm] -> bf16 copy; clears the pending set
int launch_commit(ttt_ctx* ctx, cudaStream_t s);
// W2[:, o] *= n0[o] / (||W2[:, o]|| + 1e-5) from `nblk` per-head partial column sums of squares in colsq
int launch_renorm_w2(ttt_ctx* ctx, int nblk, cudaStream_t s);
// loss[h] = sum_{r in [0, n)} loss_part[r][h]  (fixed order)
int launch_loss_reduce(ttt_ctx* ctx, int n, float* loss, cudaStream_t s);

// --- tensor-core Newton-Schulz (ns_tc.cu) ---------------------------------------------------------
int ns_tc_supported(const ttt_config* cfg);
// NS((G_valid ? G : 0) + sum partials) for all 3*nh matrices; fuse_commit: W <- W - NS(.) and the
// pending set is cleared, else the result is left in G (G_valid)
int launch_ns_tc(ttt_ctx* ctx, bool fuse_commit, cudaStream_t s);
// hd = 128: one thread-block cluster per matrix (ns_tc_wide.cu); reached through the two calls above
int ns_tc_wide_supported(const ttt_config* cfg);
int launch_ns_tc_wide(ttt_ctx* ctx, bool fuse_commit, cudaStream_t s);

// --- f32 path (f32_path.cu) ---------------------------------------------------------------------
// appends partial-gradient sets [n_partials, n_partials + used); writes loss_part rows [0, loss_rows)
int f32_accumulate(ttt_ctx* ctx, const float* K, const float* V, const float* lr, int64_t M,
                   int64_t ld, bool want_loss, int* used, int* loss_rows, cudaStream_t s);
int f32_apply(ttt_ctx* ctx, const float* Q, float* O, int64_t M, int64_t ld, cudaStream_t s);
int f32_partials_needed(const ttt_ctx* ctx, int64_t M);

// --- bf16 tensor-core path (bf16_update.cu / bf16_apply.cu) -------------------------------------
// fuse_commit: also apply W <- W - gradient inside the kernel (plain update, nothing pending);
// returns 1 (instead of TTT_OK) when it did, negative on error
int bf16_accumulate(ttt_ctx* ctx, const __nv_bfloat16* K, const __nv_bfloat16* V, const float* lr,
                    int64_t M, int64_t ld, bool want_loss, bool fuse_commit, int* used,
                    int* loss_rows, cudaStream_t s);
int bf16_apply(ttt_ctx* ctx, const __nv_bfloat16* Q, __nv_bfloat16* O, int64_t M, int64_t ld,
               cudaStream_t s);
int bf16_partials_needed(const ttt_ctx* ctx, int64_t M);
int bf16_supported(const ttt_config* cfg, char* why, size_t why_len);
// 1 if a tcgen05 kernel covers the shape, 0 if bf16 I/O must go through the fp32 CUDA-core path
int bf16_update_tensor_path(const ttt_config* cfg);
int bf16_apply_tensor_path(const ttt_config* cfg);
// hd = 128 apply kernel on CTA pairs (bf16_apply_wide_pair.cu)
int bf16_apply_wide_supported(const ttt_config* cfg);
int bf16_apply_wide_pair(ttt_ctx* ctx, const __nv_bfloat16* Q, __nv_bfloat16* O, int64_t M, int64_t ld,
                         cudaStream_t s);
// hd = 128 update kernel (bf16_update_wide.cu)
int bf16_update_wide_supported(const ttt_config* cfg);
int bf16_accumulate_wide(ttt_ctx* ctx, const __nv_bfloat16* K, const __nv_bfloat16* V, const float* lr,
                         int64_t M, int64_t ld, bool want_loss, int* used, int* loss_rows,
                         cudaStream_t s);
int bf16_wide_partials_needed(const ttt_ctx* ctx, int64_t M);
// large-dimension path (bf16_large.cu): hd a multiple of 256, plain update
int bf16_large_supported(const ttt_config* cfg);
int64_t bf16_large_loss_rows(const ttt_config* cfg);
int bf16_large_accumulate(ttt_ctx* ctx, const __nv_bfloat16* K, const __nv_bfloat16* V, const float* lr,
                          int64_t M, int64_t ld, bool want_loss, int* loss_rows, cudaStream_t s);
int bf16_large_apply(ttt_ctx* ctx, const __nv_bfloat16* Q, __nv_bfloat16* O, int64_t M, int64_t ld,
                     cudaStream_t s);
// strided bf16 [M][cols] (row stride ld) <-> dense fp32 [M][cols]
int launch_bf16_to_f32(ttt_ctx* ctx, const __nv_bfloat16* src, int64_t ld, float* dst, int64_t M, cudaStream_t s);
int launch_f32_to_bf16(ttt_ctx* ctx, const float* src, __nv_bfloat16* dst, int64_t ld, int64_t M, cudaStream_t s);

}  // namespace ttt

#define TTT_CUDA_TRY(ctx, call, what)                                   \
  do {                                                                  \
    cudaError_t e__ = (call);                                           \
    if (e__ != cudaSuccess) return ttt::set_error((ctx), TTT_ERR_CUDA, (what), e__); \
  } while (0)

#define TTT_LAUNCH_CHECK(ctx, what)                                     \
  do {                                                                  \
    cudaError_t e__ = cudaGetLastError();                               \
    if (e__ != cudaSuccess) return ttt::set_error((ctx), TTT_ERR_CUDA, (what), e__); \
    (ctx)->launches += 1;                                               \
  } while (0)
