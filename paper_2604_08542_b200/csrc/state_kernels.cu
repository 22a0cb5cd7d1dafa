// state_kernels.cu — kernels that own the fast-weight state: load/transpose at ttt_init, the
// fixed-order reduction of partial gradients, the Newton-Schulz orthonormalisation, the weight
// commit W <- W - G (Eq. 8) with optional fan-in re-normalisation, and the bf16
// operand refresh. All fp32 FFMA; the state is a few MB and L2-resident, so these kernels are
// latency/L2-bound, not HBM-bound.
#include <math.h>
#include <stdio.h>

#include "ttt_internal.h"

namespace ttt {

int set_error(ttt_ctx* ctx, int status, const char* what, cudaError_t e) {
  if (ctx) {
    if (e != cudaSuccess)
      snprintf(ctx->err, sizeof(ctx->err), "%s: %s", what, cudaGetErrorString(e));
    else
      snprintf(ctx->err, sizeof(ctx->err), "%s", what);
  }
  return status;
}

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// ------------------------------------------------------------------------------------------------
// ttt_init: user layout -> hidden-major masters + bf16 copies + initial fan-in norms.
// grid (ceil(H/32), nh, 3), block (32, 8). A 32x32 smem tile transposes W1/W3 ([hd][H] -> [H][hd]).
// ------------------------------------------------------------------------------------------------
__global__ void init_load_kernel(const float* __restrict__ W1, const float* __restrict__ W2,
                                 const float* __restrict__ W3, float* __restrict__ Wm,
                                 __nv_bfloat16* __restrict__ Wb, int nh, int hd, int H) {
  __shared__ float tile[32][33];
  const int mat = blockIdx.z, h = blockIdx.y, j0 = blockIdx.x * 32;
  const size_t me = (size_t)nh * H * hd;
  float* dst = Wm + mat * me + (size_t)h * H * hd;
  __nv_bfloat16* dstb = Wb + mat * me + (size_t)h * H * hd;
  if (mat == 1) {  // W2 [H][hd]: straight copy
    const float* src = W2 + (size_t)h * H * hd;
    for (int r = threadIdx.y; r < 32; r += blockDim.y) {
      int j = j0 + r;
      if (j >= H) break;
      for (int i = threadIdx.x; i < hd; i += 32) {
        float v = src[(size_t)j * hd + i];
        dst[(size_t)j * hd + i] = v;
        dstb[(size_t)j * hd + i] = __float2bfloat16_rn(v);
      }
    }
    return;
  }
  const float* src = (mat == 0 ? W1 : W3) + (size_t)h * hd * H;  // [hd][H]
  for (int i0 = 0; i0 < hd; i0 += 32) {
    for (int r = threadIdx.y; r < 32; r += blockDim.y) {
      int i = i0 + r, j = j0 + threadIdx.x;
      tile[r][threadIdx.x] = (i < hd && j < H) ? src[(size_t)i * H + j] : 0.f;
    }
    __syncthreads();
    for (int r = threadIdx.y; r < 32; r += blockDim.y) {
      int j = j0 + r, i = i0 + threadIdx.x;
      if (j < H && i < hd) {
        float v = tile[threadIdx.x][r];
        dst[(size_t)j * hd + i] = v;
        dstb[(size_t)j * hd + i] = __float2bfloat16_rn(v);
      }
    }
    __syncthreads();
  }
}

// initial fan-in norms. grid (nh, 3), block 256.
//   mat 0/2: n0[h][j] = || Wm[mat][h][j][:] ||   (row norm, length hd)
//   mat 1  : n0[h][o] = || Wm[1][h][:][o]   ||   (column norm, length H)
__global__ void init_norms_kernel(const float* __restrict__ Wm, float* __restrict__ n0, int nh,
                                  int hd, int H) {
  const int h = blockIdx.x, mat = blockIdx.y;
  const size_t me = (size_t)nh * H * hd;
  const float* W = Wm + mat * me + (size_t)h * H * hd;
  float* out = n0 + (mat == 0 ? (size_t)h * H
                              : mat == 1 ? (size_t)nh * H + (size_t)h * hd
                                         : (size_t)nh * H + (size_t)nh * hd + (size_t)h * H);
  if (mat == 1) {
    for (int o = threadIdx.x; o < hd; o += blockDim.x) {
      float acc = 0.f;
      for (int j = 0; j < H; ++j) { float v = W[(size_t)j * hd + o]; acc = fmaf(v, v, acc); }
      out[o] = sqrtf(acc);
    }
  } else {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nw = blockDim.x >> 5;
    for (int j = warp; j < H; j += nw) {
      float acc = 0.f;
      for (int i = lane; i < hd; i += 32) { float v = W[(size_t)j * hd + i]; acc = fmaf(v, v, acc); }
      acc = warp_sum(acc);
      if (lane == 0) out[j] = sqrtf(acc);
    }
  }
}

// ttt_get_weights: hidden-major masters -> user layout. Same tiling as init_load_kernel.
__global__ void get_weights_kernel(const float* __restrict__ Wm, float* __restrict__ W1,
                                   float* __restrict__ W2, float* __restrict__ W3, int nh, int hd,
                                   int H) {
  __shared__ float tile[32][33];
  const int mat = blockIdx.z, h = blockIdx.y, j0 = blockIdx.x * 32;
  const size_t me = (size_t)nh * H * hd;
  const float* src = Wm + mat * me + (size_t)h * H * hd;
  if (mat == 1) {
    float* dst = W2 + (size_t)h * H * hd;
    for (int r = threadIdx.y; r < 32; r += blockDim.y) {
      int j = j0 + r;
      if (j >= H) break;
      for (int i = threadIdx.x; i < hd; i += 32) dst[(size_t)j * hd + i] = src[(size_t)j * hd + i];
    }
    return;
  }
  float* dst = (mat == 0 ? W1 : W3) + (size_t)h * hd * H;
  for (int i0 = 0; i0 < hd; i0 += 32) {
    for (int r = threadIdx.y; r < 32; r += blockDim.y) {
      int j = j0 + r, i = i0 + threadIdx.x;
      tile[r][threadIdx.x] = (j < H && i < hd) ? src[(size_t)j * hd + i] : 0.f;
    }
    __syncthreads();
    for (int r = threadIdx.y; r < 32; r += blockDim.y) {
      int i = i0 + r, j = j0 + threadIdx.x;
      if (i < hd && j < H) dst[(size_t)i * H + j] = tile[threadIdx.x][r];
    }
    __syncthreads();
  }
}

// ------------------------------------------------------------------------------------------------
// fixed-order reduction of the pending partial-gradient sets into the dense gradient G
//   G[e] = (use_G ? G[e] : 0) + P[0][e] + P[1][e] + ...      (deterministic: fixed summation order)
// ------------------------------------------------------------------------------------------------
__global__ void reduce_partials_kernel(float* __restrict__ G, const float* __restrict__ P,
                                       int n_sets, size_t set_elems, int use_G) {
  size_t e = ((size_t)blockIdx.x * blockDim.x + threadIdx.x) * 4;
  if (e >= set_elems) return;
  float4 acc = use_G ? *reinterpret_cast<const float4*>(G + e) : make_float4(0.f, 0.f, 0.f, 0.f);
  for (int s = 0; s < n_sets; ++s) {
    float4 p = *reinterpret_cast<const float4*>(P + (size_t)s * set_elems + e);
    acc.x += p.x; acc.y += p.y; acc.z += p.z; acc.w += p.w;
  }
  *reinterpret_cast<float4*>(G + e) = acc;
}

__global__ void loss_reduce_kernel(const float* __restrict__ part, int n, int nh,
                                   float* __restrict__ loss) {
  int h = blockIdx.x * blockDim.x + threadIdx.x;
  if (h >= nh) return;
  float acc = 0.f;
  for (int s = 0; s < n; ++s) acc += part[(size_t)s * nh + h];
  loss[h] = acc;
}

// ------------------------------------------------------------------------------------------------
// Newton-Schulz orthonormalisation of each [H][hd] gradient matrix, in place (DESIGN.md R-NS):
//   X0 = G / (||G||_F + 1e-7);  n times:  A = X^T X (hd x hd);  B = b A + c A A;  X = a X + X B
// (the tall form of  A = X X^T; X = a X + (b A + c A^2) X  applied to G^T; NS(G^T) = NS(G)^T).
// One CTA per (matrix, head); fp32 FFMA; Gram/poly matrices in shared memory; X streamed from L2.
// Requires H >= hd (k >= 1).
// ------------------------------------------------------------------------------------------------
constexpr int NS_THREADS = 512;
constexpr int NS_ROWS = 32;  // rows of X staged per step

__global__ void __launch_bounds__(NS_THREADS, 1)
newton_schulz_kernel(float* __restrict__ G, int H, int hd, int iters) {
  extern __shared__ float ns_smem[];
  const int p = hd, pp = hd + 1;
  float* A = ns_smem;                    // [p][pp]
  float* B = A + (size_t)p * pp;         // [p][pp]
  float* Xs = B + (size_t)p * pp;        // [NS_ROWS][pp]
  float* red = Xs + (size_t)NS_ROWS * pp;  // [NS_THREADS/32]
  __shared__ float s_scale;
  float* X = G + (size_t)blockIdx.x * H * hd;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const float ca = 3.4445f, cb = -4.7750f, cc = 2.0315f;

  // Frobenius norm (fixed order: per-thread strided, warp tree, then warps in order)
  float acc = 0.f;
  for (int e = tid; e < H * hd; e += NS_THREADS) { float v = X[e]; acc = fmaf(v, v, acc); }
  acc = warp_sum(acc);
  if (lane == 0) red[warp] = acc;
  __syncthreads();
  if (tid == 0) {
    float t = 0.f;
    for (int w = 0; w < NS_THREADS / 32; ++w) t += red[w];
    s_scale = 1.0f / (sqrtf(t) + 1e-7f);
  }
  __syncthreads();
  const float scale = s_scale;
  for (int e = tid; e < H * hd; e += NS_THREADS) X[e] *= scale;
  __syncthreads();

  for (int it = 0; it < iters; ++it) {
    // A = X^T X, accumulated over row blocks
    for (int e = tid; e < p * p; e += NS_THREADS) A[(e / p) * pp + (e % p)] = 0.f;
    for (int r0 = 0; r0 < H; r0 += NS_ROWS) {
      __syncthreads();
      for (int e = tid; e < NS_ROWS * p; e += NS_THREADS) {
        int r = e / p, i = e % p;
        Xs[r * pp + i] = (r0 + r < H) ? X[(size_t)(r0 + r) * hd + i] : 0.f;
      }
      __syncthreads();
      for (int e = tid; e < p * p; e += NS_THREADS) {
        int i = e / p, i2 = e % p;
        float a = A[i * pp + i2];
#pragma unroll 8
        for (int r = 0; r < NS_ROWS; ++r) a = fmaf(Xs[r * pp + i], Xs[r * pp + i2], a);
        A[i * pp + i2] = a;
      }
    }
    __syncthreads();
    // B = b A + c A A
    for (int e = tid; e < p * p; e += NS_THREADS) {
      int i = e / p, i2 = e % p;
      float a2 = 0.f;
      for (int k = 0; k < p; ++k) a2 = fmaf(A[i * pp + k], A[k * pp + i2], a2);
      B[i * pp + i2] = cb * A[i * pp + i2] + cc * a2;
    }
    __syncthreads();
    // X = a X + X B, row block by row block
    for (int r0 = 0; r0 < H; r0 += NS_ROWS) {
      for (int e = tid; e < NS_ROWS * p; e += NS_THREADS) {
        int r = e / p, i = e % p;
        Xs[r * pp + i] = (r0 + r < H) ? X[(size_t)(r0 + r) * hd + i] : 0.f;
      }
      __syncthreads();
      for (int e = tid; e < NS_ROWS * p; e += NS_THREADS) {
        int r = e / p, i2 = e % p;
        if (r0 + r < H) {
          float xb = 0.f;
          for (int k = 0; k < p; ++k) xb = fmaf(Xs[r * pp + k], B[k * pp + i2], xb);
          X[(size_t)(r0 + r) * hd + i2] = fmaf(ca, Xs[r * pp + i2], xb);
        }
      }
      __syncthreads();
    }
  }
}

// ------------------------------------------------------------------------------------------------
// commit: W <- W - g,  g = (use_G ? G : 0) + sum_s P[s]   (Eq. 8), fp32 master + bf16 copy.
// grid (ceil(H/CM_ROWS), nh, 3), block 256 (8 warps, one row of hd per warp at a time).
// renorm (DESIGN.md R-RENORM): mats 0/2 scale each row to its initial norm here; mat 1 (column
// fan-in) writes per-block column sums of squares and is finished by renorm_w2_kernel.
// ------------------------------------------------------------------------------------------------
constexpr int CM_ROWS = 16;

__global__ void __launch_bounds__(256)
commit_kernel(float* __restrict__ Wm, __nv_bfloat16* __restrict__ Wb, const float* __restrict__ G,
              const float* __restrict__ P, int n_sets, int use_G, const float* __restrict__ n0,
              float* __restrict__ colsq, int renorm, int nh, int hd, int H) {
  __shared__ float cs[8][128];
  const int mat = blockIdx.z, h = blockIdx.y, j0 = blockIdx.x * CM_ROWS;
  const size_t me = (size_t)nh * H * hd, set = 3 * me;
  const size_t base = mat * me + (size_t)h * H * hd;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const float* n0m = n0 + (mat == 0 ? (size_t)h * H
                                    : (size_t)nh * H + (size_t)nh * hd + (size_t)h * H);
  float colacc[4] = {0.f, 0.f, 0.f, 0.f};  // hd <= 128: lane owns columns lane + 32*c
  for (int r = warp; r < CM_ROWS; r += 8) {
    const int j = j0 + r;
    if (j >= H) break;
    const size_t row = base + (size_t)j * hd;
    float w[4];
    float sq = 0.f;
#pragma unroll
    for (int c = 0; c < 4; ++c) {
      const int i = lane + 32 * c;
      w[c] = 0.f;
      if (i < hd) {
        float g = use_G ? G[row + i] : 0.f;
        for (int s = 0; s < n_sets; ++s) g += P[(size_t)s * set + row + i];
        w[c] = Wm[row + i] - g;
        sq = fmaf(w[c], w[c], sq);
      }
    }
    if (renorm && mat != 1) {
      sq = warp_sum(sq);
      const float f = n0m[j] / (sqrtf(sq) + 1e-5f);
#pragma unroll
      for (int c = 0; c < 4; ++c) w[c] *= f;
    }
#pragma unroll
    for (int c = 0; c < 4; ++c) {
      const int i = lane + 32 * c;
      if (i < hd) {
        Wm[row + i] = w[c];
        Wb[row + i] = __float2bfloat16_rn(w[c]);
        colacc[c] = fmaf(w[c], w[c], colacc[c]);
      }
    }
  }
  if (renorm && mat == 1) {
#pragma unroll
    for (int c = 0; c < 4; ++c) cs[warp][lane + 32 * c] = colacc[c];
    __syncthreads();
    for (int i = threadIdx.x; i < hd; i += blockDim.x) {
      float t = 0.f;
      for (int w8 = 0; w8 < 8; ++w8) t += cs[w8][i];
      colsq[((size_t)h * gridDim.x + blockIdx.x) * hd + i] = t;
    }
  }
}

// W2[:, o] *= n0[o] / (||W2[:, o]|| + 1e-5), norms from the per-block partial sums (fixed order).
// grid (ceil(H/CM_ROWS), nh), block 256.
__global__ void __launch_bounds__(256)
renorm_w2_kernel(float* __restrict__ Wm, __nv_bfloat16* __restrict__ Wb,
                 const float* __restrict__ colsq, const float* __restrict__ n0, int nblk, int nh,
                 int hd, int H) {
  __shared__ float f[128];
  const int h = blockIdx.y, j0 = blockIdx.x * CM_ROWS;
  const size_t me = (size_t)nh * H * hd;
  for (int i = threadIdx.x; i < hd; i += blockDim.x) {
    float t = 0.f;
    for (int b = 0; b < nblk; ++b) t += colsq[((size_t)h * nblk + b) * hd + i];
    f[i] = n0[(size_t)nh * H + (size_t)h * hd + i] / (sqrtf(t) + 1e-5f);
  }
  __syncthreads();
  const size_t base = me + (size_t)h * H * hd;
  for (int e = threadIdx.x; e < CM_ROWS * hd; e += blockDim.x) {
    const int j = j0 + e / hd, i = e % hd;
    if (j < H) {
      const float w = Wm[base + (size_t)j * hd + i] * f[i];
      Wm[base + (size_t)j * hd + i] = w;
      Wb[base + (size_t)j * hd + i] = __float2bfloat16_rn(w);
    }
  }
}

// ------------------------------------------------------------------------------------------------
// launchers
// ------------------------------------------------------------------------------------------------
int launch_init(ttt_ctx* ctx, const float* W1, const float* W2, const float* W3, cudaStream_t s) {
  const ttt_config& c = ctx->cfg;
  dim3 grid((c.hidden + 31) / 32, c.nh, 3), block(32, 8);
  init_load_kernel<<<grid, block, 0, s>>>(W1, W2, W3, ctx->Wm, ctx->Wb, c.nh, c.hd, c.hidden);
  TTT_LAUNCH_CHECK(ctx, "init_load_kernel");
  init_norms_kernel<<<dim3(c.nh, 3), 256, 0, s>>>(ctx->Wm, ctx->n0, c.nh, c.hd, c.hidden);
  TTT_LAUNCH_CHECK(ctx, "init_norms_kernel");
  return TTT_OK;
}

int launch_get_weights(ttt_ctx* ctx, float* W1, float* W2, float* W3, cudaStream_t s) {
  const ttt_config& c = ctx->cfg;
  dim3 grid((c.hidden + 31) / 32, c.nh, 3), block(32, 8);
  get_weights_kernel<<<grid, block, 0, s>>>(ctx->Wm, W1, W2, W3, c.nh, c.hd, c.hidden);
  TTT_LAUNCH_CHECK(ctx, "get_weights_kernel");
  return TTT_OK;
}

int launch_reduce_pending(ttt_ctx* ctx, cudaStream_t s) {
  const size_t set = 3 * ctx->mat_elems;
  if (ctx->n_partials == 0 && ctx->G_valid) return TTT_OK;
  const int threads = 256;
  const unsigned blocks = (unsigned)((set / 4 + threads - 1) / threads);
  reduce_partials_kernel<<<blocks, threads, 0, s>>>(ctx->G, ctx->partials, ctx->n_partials, set,
                                                    ctx->G_valid ? 1 : 0);
  TTT_LAUNCH_CHECK(ctx, "reduce_partials_kernel");
  ctx->G_valid = true;
  ctx->n_partials = 0;
  return TTT_OK;
}

int launch_loss_reduce(ttt_ctx* ctx, int n, float* loss, cudaStream_t s) {
  const int nh = ctx->cfg.nh;
  loss_reduce_kernel<<<(nh + 63) / 64, 64, 0, s>>>(ctx->loss_part, n, nh, loss);
  TTT_LAUNCH_CHECK(ctx, "loss_reduce_kernel");
  return TTT_OK;
}

int launch_commit(ttt_ctx* ctx, cudaStream_t s) {
  const ttt_config& c = ctx->cfg;
  if (c.ns_iters > 0) {
    int rc = launch_reduce_pending(ctx, s);
    if (rc != TTT_OK) return rc;
    const size_t smem = ((size_t)2 * c.hd * (c.hd + 1) + (size_t)NS_ROWS * (c.hd + 1) +
                         NS_THREADS / 32) * sizeof(float);
    static bool attr_set = false;
    if (!attr_set) {
      TTT_CUDA_TRY(ctx, cudaFuncSetAttribute(newton_schulz_kernel,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             200 * 1024), "newton_schulz smem attr");
      attr_set = true;
    }
    // linear test mode: only mat 0 carries a gradient (mats 1, 2 are identically zero)
    const int n_mats = c.linear_fast_weight ? c.nh : 3 * c.nh;
    newton_schulz_kernel<<<n_mats, NS_THREADS, smem, s>>>(ctx->G, c.hidden, c.hd, c.ns_iters);
    TTT_LAUNCH_CHECK(ctx, "newton_schulz_kernel");
  }
  const int nblk = (c.hidden + CM_ROWS - 1) / CM_ROWS;
  commit_kernel<<<dim3(nblk, c.nh, 3), 256, 0, s>>>(ctx->Wm, ctx->Wb, ctx->G, ctx->partials,
                                                    ctx->n_partials, ctx->G_valid ? 1 : 0, ctx->n0,
                                                    ctx->colsq, c.renorm, c.nh, c.hd, c.hidden);
  TTT_LAUNCH_CHECK(ctx, "commit_kernel");
  if (c.renorm) {
    renorm_w2_kernel<<<dim3(nblk, c.nh), 256, 0, s>>>(ctx->Wm, ctx->Wb, ctx->colsq, ctx->n0, nblk,
                                                      c.nh, c.hd, c.hidden);
    TTT_LAUNCH_CHECK(ctx, "renorm_w2_kernel");
  }
  ctx->G_valid = false;
  ctx->n_partials = 0;
  return TTT_OK;
}

}  // namespace ttt
