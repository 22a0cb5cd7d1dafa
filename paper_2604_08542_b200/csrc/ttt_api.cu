// ttt_api.cu — the C ABI of include/ttt.h: argument validation, context life cycle and the launch
// chains. No arithmetic here; every step of the path runs in the kernels of the other files.
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <new>

#include "ttt_internal.h"

using namespace ttt;

namespace {

thread_local char g_create_err[256] = "";

int create_fail(int status, const char* fmt, long long a = 0, long long b = 0) {
  snprintf(g_create_err, sizeof(g_create_err), fmt, a, b);
  return status;
}

// makes the context's device current for the duration of an entry point
struct DeviceGuard {
  int prev = -1, want;
  explicit DeviceGuard(const ttt_ctx* ctx) : want(ctx->cfg.device) {
    if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
    if (prev != want) cudaSetDevice(want);
  }
  ~DeviceGuard() {
    if (prev >= 0 && prev != want) cudaSetDevice(prev);
  }
};

int fail(ttt_ctx* ctx, int status, const char* fmt, long long a = 0, long long b = 0) {
  if (ctx) snprintf(ctx->err, sizeof(ctx->err), fmt, a, b);
  return status;
}

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

size_t elt_size(const ttt_ctx* ctx) { return ctx->cfg.act_dtype == TTT_BF16 ? 2 : 4; }

int check_tokens(ttt_ctx* ctx, int64_t M, int64_t ld) {
  if (M < 0) return fail(ctx, TTT_ERR_ARG, "M = %lld is negative", M);
  if (M > ctx->cfg.max_tokens)
    return fail(ctx, TTT_ERR_SHAPE, "M = %lld exceeds max_tokens = %lld", M, ctx->cfg.max_tokens);
  if (ld < (int64_t)ctx->cfg.nh * ctx->cfg.hd)
    return fail(ctx, TTT_ERR_SHAPE, "ld = %lld is smaller than nh*hd = %lld", ld,
                (long long)ctx->cfg.nh * ctx->cfg.hd);
  if ((ld * (int64_t)elt_size(ctx)) % 16 != 0)
    return fail(ctx, TTT_ERR_ALIGN, "ld*sizeof(elt) = %lld is not a multiple of 16",
                ld * (long long)elt_size(ctx));
  return TTT_OK;
}

// commit_now: the caller will commit right after (ttt_update / ttt_chunk_step); returns 1 if the
// accumulate kernel has already committed (fused path), TTT_OK if a commit is still due
int do_accumulate(ttt_ctx* ctx, const void* K, const void* V, const float* lr, int64_t M,
                  int64_t ld, float* loss, cudaStream_t s, bool commit_now = false) {
  const bool bf16 = ctx->cfg.act_dtype == TTT_BF16 && !ctx->upd_via_f32;
  if (ctx->upd_via_f32) {      // bf16 I/O on the fp32 CUDA-core path: convert K, V first
    const int64_t d = (int64_t)ctx->cfg.nh * ctx->cfg.hd;
    int rc = launch_bf16_to_f32(ctx, static_cast<const __nv_bfloat16*>(K), ld, ctx->stage[0], M, s);
    if (rc == TTT_OK) rc = launch_bf16_to_f32(ctx, static_cast<const __nv_bfloat16*>(V), ld, ctx->stage[1], M, s);
    if (rc != TTT_OK) return rc;
    K = ctx->stage[0]; V = ctx->stage[1]; ld = d;
  }
  if (ctx->large) {                  // hd >= 256: forward + gradient GEMMs, dense pending gradient
    int loss_rows = 0;
    int rc = bf16_large_accumulate(ctx, static_cast<const __nv_bfloat16*>(K), static_cast<const __nv_bfloat16*>(V),
                                   lr, M, ld, loss != nullptr, &loss_rows, s);
    if (rc == TTT_OK && loss != nullptr) rc = launch_loss_reduce(ctx, loss_rows, loss, s);
    return rc;
  }
  const int need = bf16 ? bf16_partials_needed(ctx, M) : f32_partials_needed(ctx, M);
  if (need > ctx->cap_partials)
    return fail(ctx, TTT_ERR_SHAPE, "internal: %lld partial sets needed, capacity %lld", need,
                ctx->cap_partials);
  if (ctx->n_partials + need > ctx->cap_partials) {  // fold the pending sets into G first
    int rc = launch_reduce_pending(ctx, s);
    if (rc != TTT_OK) return rc;
  }
  int used = 0, loss_rows = 0, rc;
  const bool fuse = commit_now && bf16 && ctx->cfg.ns_iters == 0 &&
                    ctx->n_partials == 0 && !ctx->G_valid;
  if (bf16)
    rc = bf16_accumulate(ctx, static_cast<const __nv_bfloat16*>(K),
                         static_cast<const __nv_bfloat16*>(V), lr, M, ld, loss != nullptr, fuse,
                         &used, &loss_rows, s);
  else
    rc = f32_accumulate(ctx, static_cast<const float*>(K), static_cast<const float*>(V), lr, M, ld,
                        loss != nullptr, &used, &loss_rows, s);
  if (rc < 0) return rc;
  const int committed = rc;
  ctx->n_partials += used;
  if (loss != nullptr) {
    rc = launch_loss_reduce(ctx, loss_rows, loss, s);
    if (rc != TTT_OK) return rc;
  }
  return committed;
}

int do_apply(ttt_ctx* ctx, const void* Q, void* O, int64_t M, int64_t ld, cudaStream_t s) {
  if (ctx->app_via_f32) {
    const int64_t d = (int64_t)ctx->cfg.nh * ctx->cfg.hd;
    int rc = launch_bf16_to_f32(ctx, static_cast<const __nv_bfloat16*>(Q), ld, ctx->stage[0], M, s);
    if (rc == TTT_OK) rc = f32_apply(ctx, ctx->stage[0], ctx->stage[1], M, d, s);
    if (rc == TTT_OK) rc = launch_f32_to_bf16(ctx, ctx->stage[1], static_cast<__nv_bfloat16*>(O), ld, M, s);
    return rc;
  }
  if (ctx->large)
    return bf16_large_apply(ctx, static_cast<const __nv_bfloat16*>(Q), static_cast<__nv_bfloat16*>(O), M, ld, s);
  if (ctx->cfg.act_dtype == TTT_BF16)
    return bf16_apply(ctx, static_cast<const __nv_bfloat16*>(Q), static_cast<__nv_bfloat16*>(O), M,
                      ld, s);
  return f32_apply(ctx, static_cast<const float*>(Q), static_cast<float*>(O), M, ld, s);
}

int check_update_args(ttt_ctx* ctx, const void* K, const void* V, const float* lr, int64_t M,
                      int64_t ld) {
  if (!ctx->initialised) return fail(ctx, TTT_ERR_STATE, "ttt_init has not been called");
  int rc = check_tokens(ctx, M, ld);
  if (rc != TTT_OK) return rc;
  if (M == 0) return TTT_OK;
  if (!K || !V || !lr) return fail(ctx, TTT_ERR_ARG, "K, V and lr must not be NULL");
  if (!aligned16(K) || !aligned16(V))
    return fail(ctx, TTT_ERR_ALIGN, "K and V must be 16-byte aligned");
  return TTT_OK;
}

int check_apply_args(ttt_ctx* ctx, const void* Q, const void* O, int64_t M, int64_t ld) {
  if (!ctx->initialised) return fail(ctx, TTT_ERR_STATE, "ttt_init has not been called");
  int rc = check_tokens(ctx, M, ld);
  if (rc != TTT_OK) return rc;
  if (M == 0) return TTT_OK;
  if (!Q || !O) return fail(ctx, TTT_ERR_ARG, "Q and O must not be NULL");
  if (Q == O) return fail(ctx, TTT_ERR_ARG, "O must not alias Q");
  if (!aligned16(Q) || !aligned16(O))
    return fail(ctx, TTT_ERR_ALIGN, "Q and O must be 16-byte aligned");
  return TTT_OK;
}

}  // namespace

extern "C" {

int ttt_create(ttt_ctx** out, const ttt_config* cfg) {
  g_create_err[0] = 0;
  if (!out || !cfg) return create_fail(TTT_ERR_ARG, "out and cfg must not be NULL");
  if (cfg->nh < 1 || cfg->hd < 1 || cfg->hidden < 1 || cfg->max_tokens < 1 || cfg->ns_iters < 0 ||
      (cfg->renorm != 0 && cfg->renorm != 1) ||
      (cfg->linear_fast_weight != 0 && cfg->linear_fast_weight != 1) ||
      (cfg->cuda_core_fallback != 0 && cfg->cuda_core_fallback != 1) || cfg->reserved != 0 ||
      (cfg->act_dtype != TTT_F32 && cfg->act_dtype != TTT_BF16))
    return create_fail(TTT_ERR_ARG, "a ttt_config field is out of range");
  if (cfg->hd % 4 != 0 || cfg->hidden % 4 != 0 || (cfg->hd > 128 && !bf16_large_supported(cfg)))
    return create_fail(TTT_ERR_SHAPE, "hd = %lld, hidden = %lld: both must be multiples of 4 and hd <= 128 (bf16 "
                       "without Newton-Schulz / renorm also: hd a multiple of 256 up to 2048, hidden a multiple of 128)",
                       cfg->hd, cfg->hidden);
  if (cfg->linear_fast_weight && cfg->hidden != cfg->hd)
    return create_fail(TTT_ERR_SHAPE, "linear test mode needs hidden == hd");
  if (cfg->ns_iters > 0 && cfg->hidden < cfg->hd)
    return create_fail(TTT_ERR_UNSUPPORTED, "Newton-Schulz needs hidden >= hd");
  // hd 64 | 128 on the tensor path: a hidden size that is not a multiple of 128 (k = 1 at hd 64: H = 64) runs
  // as the next multiple with zero-padded hidden units
  const ttt_config* ucfg = cfg;
  ttt_config eff = *cfg;
  if (cfg->act_dtype == TTT_BF16 && !cfg->cuda_core_fallback && !cfg->linear_fast_weight &&
      (cfg->hd == 64 || cfg->hd == 128) && cfg->hidden % 128 != 0) {
    eff.hidden = (cfg->hidden + 127) / 128 * 128;
    if (bf16_update_tensor_path(&eff) && bf16_apply_tensor_path(&eff)) cfg = &eff;
  }
  if (cfg->act_dtype == TTT_BF16) {
    char why[200];
    if (!bf16_supported(cfg, why, sizeof(why))) return create_fail(TTT_ERR_UNSUPPORTED, why);
    if (!cfg->cuda_core_fallback && !(bf16_update_tensor_path(cfg) && bf16_apply_tensor_path(cfg)))
      return create_fail(TTT_ERR_UNSUPPORTED,
                         "bf16: no tcgen05 kernel for hd = %lld, hidden = %lld (tensor kernels: hd 64 with "
                         "hidden 128|256, hd 128 with hidden %% 128 == 0); cfg.cuda_core_fallback = 1 "
                         "selects the fp32 CUDA-core kernels", cfg->hd, cfg->hidden);
    if (!cfg->cuda_core_fallback && cfg->ns_iters > 0 && !ns_tc_supported(cfg))
      return create_fail(TTT_ERR_UNSUPPORTED, "bf16: no tensor-core Newton-Schulz kernel for hidden = %lld",
                         cfg->hidden);
  }
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || cfg->device < 0 || cfg->device >= ndev)
    return create_fail(TTT_ERR_CUDA, "device %lld does not exist", cfg->device);
  int prev_dev = -1;
  cudaGetDevice(&prev_dev);
  struct Restore { int d; ~Restore() { if (d >= 0) cudaSetDevice(d); } } restore{prev_dev};
  if (cudaSetDevice(cfg->device) != cudaSuccess) return create_fail(TTT_ERR_CUDA, "cudaSetDevice failed");
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, cfg->device) != cudaSuccess)
    return create_fail(TTT_ERR_CUDA, "cudaGetDeviceProperties failed");
  if (prop.major != 10)   // sm_100a only; no fallback
    return create_fail(TTT_ERR_UNSUPPORTED, "device has compute capability %lld.x, sm_100a is required", prop.major);

  ttt_ctx* ctx = new (std::nothrow) ttt_ctx();
  if (!ctx) return create_fail(TTT_ERR_NOMEM, "out of host memory");
  memset(ctx, 0, sizeof(*ctx));
  ctx->cfg = *cfg;
  ctx->user_hidden = ucfg->hidden;
  ctx->sm_count = prop.multiProcessorCount;
  ctx->mat_elems = (size_t)cfg->nh * cfg->hidden * cfg->hd;
  const size_t set = 3 * ctx->mat_elems;
  const bool is_bf16 = cfg->act_dtype == TTT_BF16;
  ctx->large = bf16_large_supported(cfg) != 0;
  ctx->upd_via_f32 = is_bf16 && !bf16_update_tensor_path(cfg);
  ctx->app_via_f32 = is_bf16 && !bf16_apply_tensor_path(cfg);
  const bool bf16 = is_bf16 && !ctx->upd_via_f32;          // update on the tensor cores
  const bool any_tc = is_bf16 && !(ctx->upd_via_f32 && ctx->app_via_f32);
  const bool any_f32 = !is_bf16 || ctx->upd_via_f32 || ctx->app_via_f32;
  ctx->cap_partials = 2 * (bf16 ? bf16_partials_needed(ctx, cfg->max_tokens)
                                : f32_partials_needed(ctx, cfg->max_tokens));
  if (ctx->cap_partials < 4) ctx->cap_partials = 4;
  ctx->cap_loss_rows = ctx->cap_partials * ((cfg->hidden + 127) / 128);
  if (ctx->large) ctx->cap_loss_rows = (int)bf16_large_loss_rows(cfg);
  const int nblk = (cfg->hidden + 15) / 16 + 160;   // commit row blocks, or (slices x splits) of the fused commit

  bool ok = true;
  auto alloc = [&](void** p, size_t bytes) {
    if (ok && cudaMalloc(p, bytes) != cudaSuccess) ok = false;
  };
  alloc((void**)&ctx->Wm, set * sizeof(float));
  alloc((void**)&ctx->Wb, set * sizeof(ttt_wop_t));
  if (is_bf16 && (bf16_apply_wide_supported(cfg) || ctx->large)) alloc((void**)&ctx->Wq, set * sizeof(__nv_bfloat16));
  if (ctx->large)
    for (int i = 0; i < 3; ++i)
      alloc((void**)&ctx->lact[i], (size_t)cfg->max_tokens * cfg->nh * cfg->hidden * sizeof(__nv_bfloat16));
  alloc((void**)&ctx->n0, ((size_t)2 * cfg->nh * cfg->hidden + (size_t)cfg->nh * cfg->hd) * sizeof(float));
  alloc((void**)&ctx->colsq, (size_t)cfg->nh * nblk * cfg->hd * sizeof(float));
  alloc((void**)&ctx->G, set * sizeof(float));
  alloc((void**)&ctx->partials, (ctx->large ? (size_t)4 : (size_t)ctx->cap_partials * set) * sizeof(float));
  alloc((void**)&ctx->loss_part, (size_t)ctx->cap_loss_rows * cfg->nh * sizeof(float));
  if (bf16 && !ctx->large) {
    const size_t nctr = (size_t)cfg->nh * ((cfg->hidden + 127) / 128);
    alloc((void**)&ctx->sync_ctr, nctr * sizeof(unsigned));
    if (ok && cudaMemset(ctx->sync_ctr, 0, nctr * sizeof(unsigned)) != cudaSuccess) ok = false;
  }
  if (cfg->ns_iters > 0 && ns_tc_wide_supported(cfg))
    alloc((void**)&ctx->ns_scratch, (size_t)3 * cfg->nh * (cfg->hidden / 128) * 2 * 128 * 128 * sizeof(float));
  if (ctx->upd_via_f32 || ctx->app_via_f32) {
    const size_t st = (size_t)cfg->max_tokens * cfg->nh * cfg->hd * sizeof(float);
    alloc((void**)&ctx->stage[0], st);
    alloc((void**)&ctx->stage[1], st);
  }
  if (any_f32) {
    const size_t act = (size_t)cfg->nh * cfg->max_tokens * cfg->hidden * sizeof(float);
    for (int i = 0; i < 3; ++i) alloc((void**)&ctx->act[i], act);
    alloc((void**)&ctx->loss_blk, (size_t)cfg->nh * ((cfg->max_tokens + 63) / 64) *
                                      ((cfg->hidden + 63) / 64) * sizeof(float));
  }
  if (any_tc) {
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &ctx->encode_tiled, cudaEnableDefault,
                                &qres) != cudaSuccess ||
        ctx->encode_tiled == nullptr)
      ok = false;
  }
  if (!ok) {
    cudaGetLastError();
    ttt_destroy(ctx);
    return create_fail(TTT_ERR_NOMEM, "device memory allocation failed");
  }
  *out = ctx;
  return TTT_OK;
}

const char* ttt_create_error(void) { return g_create_err; }

int ttt_kernel_path(const ttt_ctx* ctx, int* update_tc, int* apply_tc) {
  if (!ctx) return TTT_ERR_ARG;
  const bool bf16 = ctx->cfg.act_dtype == TTT_BF16;
  if (update_tc) *update_tc = bf16 && !ctx->upd_via_f32;
  if (apply_tc) *apply_tc = bf16 && !ctx->app_via_f32;
  return TTT_OK;
}

void ttt_destroy(ttt_ctx* ctx) {
  if (!ctx) return;
  DeviceGuard dg(ctx);
  cudaDeviceSynchronize();
  cudaFree(ctx->Wm); cudaFree(ctx->Wb); cudaFree(ctx->Wq); cudaFree(ctx->lact[0]); cudaFree(ctx->lact[1]); cudaFree(ctx->lact[2]); cudaFree(ctx->n0); cudaFree(ctx->colsq);
  cudaFree(ctx->G); cudaFree(ctx->partials); cudaFree(ctx->loss_part); cudaFree(ctx->loss_blk); cudaFree(ctx->sync_ctr); cudaFree(ctx->ns_scratch); cudaFree(ctx->stage[0]); cudaFree(ctx->stage[1]);
  for (int i = 0; i < 3; ++i) cudaFree(ctx->act[i]);
  delete ctx;
}

int ttt_init(ttt_ctx* ctx, const float* W1, const float* W2, const float* W3, void* stream) {
  if (!ctx) return TTT_ERR_ARG;
  if (!W1 || !W2 || !W3) return fail(ctx, TTT_ERR_ARG, "W1, W2 and W3 must not be NULL");
  DeviceGuard dg(ctx);
  int rc = launch_init(ctx, W1, W2, W3, static_cast<cudaStream_t>(stream));
  if (rc != TTT_OK) return rc;
  ctx->initialised = true;
  ctx->n_partials = 0;
  ctx->G_valid = false;
  return TTT_OK;
}

int ttt_accumulate(ttt_ctx* ctx, const void* K, const void* V, const float* lr, int64_t M,
                   int64_t ld, float* loss, void* stream) {
  if (!ctx) return TTT_ERR_ARG;
  int rc = check_update_args(ctx, K, V, lr, M, ld);
  if (rc != TTT_OK || M == 0) return rc;
  DeviceGuard dg(ctx);
  rc = do_accumulate(ctx, K, V, lr, M, ld, loss, static_cast<cudaStream_t>(stream));
  return rc < 0 ? rc : TTT_OK;
}

int ttt_commit(ttt_ctx* ctx, void* stream) {
  if (!ctx) return TTT_ERR_ARG;
  if (!ctx->initialised) return fail(ctx, TTT_ERR_STATE, "ttt_init has not been called");
  if (ctx->n_partials == 0 && !ctx->G_valid) return TTT_OK;  // nothing pending
  DeviceGuard dg(ctx);
  return launch_commit(ctx, static_cast<cudaStream_t>(stream));
}

int ttt_pending_gradient(ttt_ctx* ctx, float** G, int64_t* n_elements, void* stream) {
  if (!ctx || !G || !n_elements) return TTT_ERR_ARG;
  if (!ctx->initialised) return fail(ctx, TTT_ERR_STATE, "ttt_init has not been called");
  if (ctx->n_partials == 0 && !ctx->G_valid)
    return fail(ctx, TTT_ERR_STATE, "no pending gradient (call ttt_accumulate first)");
  DeviceGuard dg(ctx);
  int rc = launch_reduce_pending(ctx, static_cast<cudaStream_t>(stream));
  if (rc != TTT_OK) return rc;
  *G = ctx->G;
  *n_elements = (int64_t)(3 * ctx->mat_elems);
  return TTT_OK;
}

int ttt_update(ttt_ctx* ctx, const void* K, const void* V, const float* lr, int64_t M, int64_t ld,
               float* loss, void* stream) {
  if (!ctx) return TTT_ERR_ARG;
  int rc = check_update_args(ctx, K, V, lr, M, ld);
  if (rc != TTT_OK || M == 0) return rc;
  DeviceGuard dg(ctx);
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  rc = do_accumulate(ctx, K, V, lr, M, ld, loss, s, true);
  if (rc < 0) return rc;
  return rc == 1 ? TTT_OK : launch_commit(ctx, s);
}

int ttt_apply(ttt_ctx* ctx, const void* Q, void* O, int64_t M, int64_t ld, void* stream) {
  if (!ctx) return TTT_ERR_ARG;
  int rc = check_apply_args(ctx, Q, O, M, ld);
  if (rc != TTT_OK || M == 0) return rc;
  DeviceGuard dg(ctx);
  return do_apply(ctx, Q, O, M, ld, static_cast<cudaStream_t>(stream));
}

int ttt_chunk_step(ttt_ctx* ctx, const void* Q, const void* K, const void* V, const float* lr,
                   void* O, int64_t M, int64_t ld, float* loss, void* stream) {
  if (!ctx) return TTT_ERR_ARG;
  int rc = check_update_args(ctx, K, V, lr, M, ld);
  if (rc != TTT_OK) return rc;
  rc = check_apply_args(ctx, Q, O, M, ld);
  if (rc != TTT_OK || M == 0) return rc;
  DeviceGuard dg(ctx);
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  rc = do_accumulate(ctx, K, V, lr, M, ld, loss, s, true);
  if (rc < 0) return rc;
  if (rc != 1) {
    rc = launch_commit(ctx, s);
    if (rc != TTT_OK) return rc;
  }
  // the kernels between here and the caller's last write of Q are this library's own: the apply
  // kernel may request its first Q tiles before its programmatic-dependency wait
  ctx->apply_q_early = 1;
  rc = do_apply(ctx, Q, O, M, ld, s);
  ctx->apply_q_early = 0;
  return rc;
}

int ttt_get_weights(ttt_ctx* ctx, float* W1, float* W2, float* W3, void* stream) {
  if (!ctx) return TTT_ERR_ARG;
  if (!ctx->initialised) return fail(ctx, TTT_ERR_STATE, "ttt_init has not been called");
  if (!W1 || !W2 || !W3) return fail(ctx, TTT_ERR_ARG, "W1, W2 and W3 must not be NULL");
  DeviceGuard dg(ctx);
  return launch_get_weights(ctx, W1, W2, W3, static_cast<cudaStream_t>(stream));
}

int64_t ttt_launch_count(const ttt_ctx* ctx) { return ctx ? ctx->launches : 0; }

const char* ttt_strerror(int status) {
  switch (status) {
    case TTT_OK: return "ok";
    case TTT_ERR_ARG: return "invalid argument";
    case TTT_ERR_SHAPE: return "shape out of range";
    case TTT_ERR_ALIGN: return "misaligned pointer or stride";
    case TTT_ERR_STATE: return "context not in the required state";
    case TTT_ERR_UNSUPPORTED: return "configuration not supported by the sm_100a kernels";
    case TTT_ERR_NOMEM: return "out of device memory";
    case TTT_ERR_CUDA: return "CUDA error";
    default: return "unknown status";
  }
}

const char* ttt_last_error(const ttt_ctx* ctx) { return ctx ? ctx->err : ""; }

const char* ttt_version(void) { return "ttt-b200 0.2 (sm_100a)"; }

}  // extern "C"
