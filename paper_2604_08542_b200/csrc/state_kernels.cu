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
// ttt_init: user layout -> hidden-major masters + bf16 copies + initial fan-in norms, fused.
// grid (ceil(H/32), nh, 3), block (32, 8): a CTA owns 32 hidden rows of one matrix. A 32x32 smem
// tile transposes W1/W3 ([hd][H] -> [H][hd]). Fan-in norms (DESIGN.md R-RENORM):
//   mat 0/2: n0[h][j] = ||row j||  (length hd)   -> finished here (a warp owns whole rows)
//   mat 1  : n0[h][o] = ||column o|| (length H)  -> per-CTA partial sums of squares to colsq,
//            finished by init_colnorm_kernel in a fixed order.
// ------------------------------------------------------------------------------------------------
__global__ void init_load_kernel(const float* __restrict__ W1, const float* __restrict__ W2,
                                 const float* __restrict__ W3, float* __restrict__ Wm,
                                 ttt_wop_t* __restrict__ Wb, __nv_bfloat16* __restrict__ Wq,
                                 float* __restrict__ n0, float* __restrict__ colsq, int nh, int hd, int H,
                                 int Hu) {   // Hu = the caller's hidden size (rows Hu .. H-1 are zero padding)
  __shared__ float tile[32][33];
  __shared__ float cs[8][128];
  const int mat = blockIdx.z, h = blockIdx.y, j0 = blockIdx.x * 32;
  const int tx = threadIdx.x, ty = threadIdx.y;
  const size_t me = (size_t)nh * H * hd;
  float* dst = Wm + mat * me + (size_t)h * H * hd;
  ttt_wop_t* dstb = Wb + mat * me + (size_t)h * H * hd;
  __nv_bfloat16* dstq = Wq ? Wq + mat * me + (size_t)h * H * hd : nullptr;
  if (mat == 1) {  // W2 [H][hd]: straight copy + column sums of squares over this CTA's rows
    const float* src = W2 + (size_t)h * Hu * hd;
    for (int cb = 0; cb < hd; cb += 128) {           // 128 columns at a time (hd > 128: the paper's shape)
      float colacc[4] = {0.f, 0.f, 0.f, 0.f};
      for (int r = ty; r < 32; r += 8) {
        const int j = j0 + r;
        if (j >= H) break;
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          const int i = cb + tx + 32 * c;
          if (i < hd) {
            const float v = j < Hu ? src[(size_t)j * hd + i] : 0.f;
            dst[(size_t)j * hd + i] = v;
            dstb[(size_t)j * hd + i] = ttt_to_wop(v);
            if (dstq) dstq[(size_t)j * hd + i] = __float2bfloat16_rn(v);
            colacc[c] = fmaf(v, v, colacc[c]);
          }
        }
      }
      __syncthreads();
#pragma unroll
      for (int c = 0; c < 4; ++c) cs[ty][tx + 32 * c] = colacc[c];
      __syncthreads();
      for (int i = ty * 32 + tx; i < 128 && cb + i < hd; i += 256) {
        float t = 0.f;
        for (int w = 0; w < 8; ++w) t += cs[w][i];
        colsq[((size_t)h * gridDim.x + blockIdx.x) * hd + cb + i] = t;
      }
    }
    return;
  }
  const float* src = (mat == 0 ? W1 : W3) + (size_t)h * hd * Hu;  // [hd][Hu]
  float rowacc[4] = {0.f, 0.f, 0.f, 0.f};                        // rows j0 + ty + 8k
  for (int i0 = 0; i0 < hd; i0 += 32) {
    for (int r = ty; r < 32; r += 8) {
      const int i = i0 + r, j = j0 + tx;
      tile[r][tx] = (i < hd && j < Hu) ? src[(size_t)i * Hu + j] : 0.f;
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const int r = ty + 8 * k, j = j0 + r, i = i0 + tx;
      if (j < H && i < hd) {
        const float v = tile[tx][r];
        dst[(size_t)j * hd + i] = v;
        dstb[(size_t)j * hd + i] = ttt_to_wop(v);
        if (dstq) dstq[(size_t)j * hd + i] = __float2bfloat16_rn(v);
        rowacc[k] = fmaf(v, v, rowacc[k]);
      }
    }
    __syncthreads();
  }
  float* out = n0 + (mat == 0 ? (size_t)h * H : (size_t)nh * H + (size_t)nh * hd + (size_t)h * H);
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    const float t = warp_sum(rowacc[k]);
    const int j = j0 + ty + 8 * k;
    if (tx == 0 && j < H) out[j] = sqrtf(t);
  }
}

// n0[h][o] of W2 from the per-CTA partial column sums of squares. grid (nh), block 128.
__global__ void init_colnorm_kernel(const float* __restrict__ colsq, float* __restrict__ n0,
                                    int nblk, int nh, int hd, int H) {
  const int h = blockIdx.x;
  for (int i = threadIdx.x; i < hd; i += blockDim.x) {
    float t = 0.f;
    for (int b = 0; b < nblk; ++b) t += colsq[((size_t)h * nblk + b) * hd + i];
    n0[(size_t)nh * H + (size_t)h * hd + i] = sqrtf(t);
  }
}

// ttt_get_weights: hidden-major masters -> user layout. Same tiling as init_load_kernel.
__global__ void get_weights_kernel(const float* __restrict__ Wm, float* __restrict__ W1,
                                   float* __restrict__ W2, float* __restrict__ W3, int nh, int hd,
                                   int H, int Hu) {
  __shared__ float tile[32][33];
  const int mat = blockIdx.z, h = blockIdx.y, j0 = blockIdx.x * 32;
  const size_t me = (size_t)nh * H * hd;
  const float* src = Wm + mat * me + (size_t)h * H * hd;
  if (mat == 1) {
    float* dst = W2 + (size_t)h * Hu * hd;
    for (int r = threadIdx.y; r < 32; r += blockDim.y) {
      int j = j0 + r;
      if (j >= Hu) break;
      for (int i = threadIdx.x; i < hd; i += 32) dst[(size_t)j * hd + i] = src[(size_t)j * hd + i];
    }
    return;
  }
  float* dst = (mat == 0 ? W1 : W3) + (size_t)h * hd * Hu;
  for (int i0 = 0; i0 < hd; i0 += 32) {
    for (int r = threadIdx.y; r < 32; r += blockDim.y) {
      int j = j0 + r, i = i0 + threadIdx.x;
      tile[r][threadIdx.x] = (j < H && i < hd) ? src[(size_t)j * hd + i] : 0.f;
    }
    __syncthreads();
    for (int r = threadIdx.y; r < 32; r += blockDim.y) {
      int i = i0 + r, j = j0 + threadIdx.x;
      if (i < hd && j < Hu) dst[(size_t)i * Hu + j] = tile[threadIdx.x][r];
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

// float4 per thread, `tpr` (power of two >= hd/4, <= 32) threads per row, 256/tpr rows per pass.
__global__ void __launch_bounds__(256)
commit_kernel(float* __restrict__ Wm, ttt_wop_t* __restrict__ Wb, __nv_bfloat16* __restrict__ Wq,
              const float* __restrict__ G,
              const float* __restrict__ P, int n_sets, int use_G, const float* __restrict__ n0,
              float* __restrict__ colsq, int renorm, int nh, int hd, int H, int tpr) {
  __shared__ float4 cs[256];
  const int mat = blockIdx.z, h = blockIdx.y, j0 = blockIdx.x * CM_ROWS;
  const size_t me = (size_t)nh * H * hd, set = 3 * me;
  const size_t base = mat * me + (size_t)h * H * hd;
  const int rows_per_pass = 256 / tpr;
  const int rr = threadIdx.x / tpr, c4 = (threadIdx.x % tpr) * 4;
  const bool col_ok = c4 < hd;
  const float* n0m = n0 + (mat == 0 ? (size_t)h * H
                                    : (size_t)nh * H + (size_t)nh * hd + (size_t)h * H);
  float4 colacc = make_float4(0.f, 0.f, 0.f, 0.f);
  for (int r = rr; r < CM_ROWS; r += rows_per_pass) {
    const int j = j0 + r;
    const bool ok = col_ok && j < H;
    const size_t e = base + (size_t)j * hd + c4;
    float4 w = make_float4(0.f, 0.f, 0.f, 0.f);
    if (ok) {
      float4 g = use_G ? *reinterpret_cast<const float4*>(G + e) : make_float4(0.f, 0.f, 0.f, 0.f);
      const float* p = P + e;
      int s = 0;
      for (; s + 4 <= n_sets; s += 4) {     // four loads in flight, summed in set order
        const float4 p0 = *reinterpret_cast<const float4*>(p + (size_t)s * set);
        const float4 p1 = *reinterpret_cast<const float4*>(p + (size_t)(s + 1) * set);
        const float4 p2 = *reinterpret_cast<const float4*>(p + (size_t)(s + 2) * set);
        const float4 p3 = *reinterpret_cast<const float4*>(p + (size_t)(s + 3) * set);
        g.x += p0.x; g.y += p0.y; g.z += p0.z; g.w += p0.w;
        g.x += p1.x; g.y += p1.y; g.z += p1.z; g.w += p1.w;
        g.x += p2.x; g.y += p2.y; g.z += p2.z; g.w += p2.w;
        g.x += p3.x; g.y += p3.y; g.z += p3.z; g.w += p3.w;
      }
      for (; s < n_sets; ++s) {
        const float4 p0 = *reinterpret_cast<const float4*>(p + (size_t)s * set);
        g.x += p0.x; g.y += p0.y; g.z += p0.z; g.w += p0.w;
      }
      const float4 w0 = *reinterpret_cast<const float4*>(Wm + e);
      w = make_float4(w0.x - g.x, w0.y - g.y, w0.z - g.z, w0.w - g.w);
    }
    if (renorm && mat != 1) {               // row fan-in: scale the row back to its initial norm
      float sq = w.x * w.x + w.y * w.y + w.z * w.z + w.w * w.w;
      for (int o = tpr >> 1; o > 0; o >>= 1) sq += __shfl_xor_sync(0xffffffffu, sq, o);
      const float f = (j < H) ? n0m[j] / (sqrtf(sq) + 1e-5f) : 0.f;
      w.x *= f; w.y *= f; w.z *= f; w.w *= f;
    }
    if (ok) {
      *reinterpret_cast<float4*>(Wm + e) = w;
      *reinterpret_cast<uint2*>(Wb + e) = make_uint2(ttt_pack_wop2(w.x, w.y), ttt_pack_wop2(w.z, w.w));
      if (Wq) {
        const __nv_bfloat162 lo = __floats2bfloat162_rn(w.x, w.y), hi = __floats2bfloat162_rn(w.z, w.w);
        *reinterpret_cast<uint2*>(Wq + e) = make_uint2(*reinterpret_cast<const uint32_t*>(&lo),
                                                        *reinterpret_cast<const uint32_t*>(&hi));
      }
      colacc.x = fmaf(w.x, w.x, colacc.x); colacc.y = fmaf(w.y, w.y, colacc.y);
      colacc.z = fmaf(w.z, w.z, colacc.z); colacc.w = fmaf(w.w, w.w, colacc.w);
    }
  }
  if (renorm && mat == 1) {                 // column fan-in: per-CTA partial sums of squares
    cs[threadIdx.x] = colacc;
    __syncthreads();
    if (threadIdx.x < tpr && col_ok) {
      float4 t = make_float4(0.f, 0.f, 0.f, 0.f);
      for (int r = 0; r < rows_per_pass; ++r) {
        const float4 v = cs[r * tpr + threadIdx.x];
        t.x += v.x; t.y += v.y; t.z += v.z; t.w += v.w;
      }
      *reinterpret_cast<float4*>(colsq + ((size_t)h * gridDim.x + blockIdx.x) * hd + c4) = t;
    }
  }
}

// W2[:, o] *= n0[o] / (||W2[:, o]|| + 1e-5), norms from the per-block partial sums (fixed order).
// grid (ceil(H/CM_ROWS), nh), block 256.
__global__ void __launch_bounds__(256)
renorm_w2_kernel(float* __restrict__ Wm, ttt_wop_t* __restrict__ Wb, __nv_bfloat16* __restrict__ Wq,
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
      Wb[base + (size_t)j * hd + i] = ttt_to_wop(w);
      if (Wq) Wq[base + (size_t)j * hd + i] = __float2bfloat16_rn(w);
    }
  }
}

// plain commit for the large-dimension path (hd > 128: no Newton-Schulz, no re-normalisation):
// W <- W - G element-wise (Eq. 8), fp32 master + fp16 and bf16 operand copies.
__global__ void __launch_bounds__(256)
commit_plain_kernel(float* __restrict__ Wm, ttt_wop_t* __restrict__ Wb, __nv_bfloat16* __restrict__ Wq,
                    const float* __restrict__ G, size_t n4) {
  const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= n4) return;
  float4 w = reinterpret_cast<const float4*>(Wm)[e];
  const float4 g = reinterpret_cast<const float4*>(G)[e];
  w.x -= g.x; w.y -= g.y; w.z -= g.z; w.w -= g.w;
  reinterpret_cast<float4*>(Wm)[e] = w;
  reinterpret_cast<uint2*>(Wb)[e] = make_uint2(ttt_pack_wop2(w.x, w.y), ttt_pack_wop2(w.z, w.w));
  if (Wq) {
    const __nv_bfloat162 lo = __floats2bfloat162_rn(w.x, w.y), hi = __floats2bfloat162_rn(w.z, w.w);
    reinterpret_cast<uint2*>(Wq)[e] = make_uint2(*reinterpret_cast<const uint32_t*>(&lo),
                                                  *reinterpret_cast<const uint32_t*>(&hi));
  }
}

// ------------------------------------------------------------------------------------------------
// launchers
// ------------------------------------------------------------------------------------------------
int launch_init(ttt_ctx* ctx, const float* W1, const float* W2, const float* W3, cudaStream_t s) {
  const ttt_config& c = ctx->cfg;
  dim3 grid((c.hidden + 31) / 32, c.nh, 3), block(32, 8);
  init_load_kernel<<<grid, block, 0, s>>>(W1, W2, W3, ctx->Wm, ctx->Wb, ctx->Wq, ctx->n0, ctx->colsq, c.nh,
                                          c.hd, c.hidden, ctx->user_hidden);
  TTT_LAUNCH_CHECK(ctx, "init_load_kernel");
  init_colnorm_kernel<<<c.nh, 128, 0, s>>>(ctx->colsq, ctx->n0, (int)grid.x, c.nh, c.hd, c.hidden);
  TTT_LAUNCH_CHECK(ctx, "init_colnorm_kernel");
  return TTT_OK;
}

int launch_get_weights(ttt_ctx* ctx, float* W1, float* W2, float* W3, cudaStream_t s) {
  const ttt_config& c = ctx->cfg;
  dim3 grid((c.hidden + 31) / 32, c.nh, 3), block(32, 8);
  get_weights_kernel<<<grid, block, 0, s>>>(ctx->Wm, W1, W2, W3, c.nh, c.hd, c.hidden, ctx->user_hidden);
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

int launch_renorm_w2(ttt_ctx* ctx, int nblk, cudaStream_t s) {
  const ttt_config& c = ctx->cfg;
  const int nrow = (c.hidden + CM_ROWS - 1) / CM_ROWS;
  renorm_w2_kernel<<<dim3(nrow, c.nh), 256, 0, s>>>(ctx->Wm, ctx->Wb, ctx->Wq, ctx->colsq, ctx->n0, nblk, c.nh,
                                                    c.hd, c.hidden);
  TTT_LAUNCH_CHECK(ctx, "renorm_w2_kernel");
  return TTT_OK;
}

int launch_commit(ttt_ctx* ctx, cudaStream_t s) {
  const ttt_config& c = ctx->cfg;
  if (ctx->large) {                       // hd > 128: the gradient GEMMs left the dense gradient in G
    const size_t n4 = 3 * ctx->mat_elems / 4;
    commit_plain_kernel<<<(unsigned)((n4 + 255) / 256), 256, 0, s>>>(ctx->Wm, ctx->Wb, ctx->Wq, ctx->G, n4);
    TTT_LAUNCH_CHECK(ctx, "commit_plain_kernel");
    ctx->G_valid = false;
    ctx->n_partials = 0;
    return TTT_OK;
  }
  if (c.ns_iters > 0 && ns_tc_supported(&c)) {
    // tensor-core NS; folds the partial sets itself and, without renorm, commits W <- W - NS(g)
    int rc = launch_ns_tc(ctx, c.renorm == 0, s);
    if (rc != TTT_OK || c.renorm == 0) return rc;
  } else if (c.ns_iters > 0) {
    int rc = launch_reduce_pending(ctx, s);
    if (rc != TTT_OK) return rc;
    const size_t smem = ((size_t)2 * c.hd * (c.hd + 1) + (size_t)NS_ROWS * (c.hd + 1) +
                         NS_THREADS / 32) * sizeof(float);
    if (!(ctx->attr_done & ATTR_NS_F32)) {
      TTT_CUDA_TRY(ctx, cudaFuncSetAttribute(newton_schulz_kernel,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             200 * 1024), "newton_schulz smem attr");
      ctx->attr_done |= ATTR_NS_F32;
    }
    // linear test mode: only mat 0 carries a gradient (mats 1, 2 are identically zero)
    const int n_mats = c.linear_fast_weight ? c.nh : 3 * c.nh;
    newton_schulz_kernel<<<n_mats, NS_THREADS, smem, s>>>(ctx->G, c.hidden, c.hd, c.ns_iters);
    TTT_LAUNCH_CHECK(ctx, "newton_schulz_kernel");
  }
  const int nblk = (c.hidden + CM_ROWS - 1) / CM_ROWS;
  int tpr = 1;
  while (tpr * 4 < c.hd) tpr <<= 1;
  commit_kernel<<<dim3(nblk, c.nh, 3), 256, 0, s>>>(ctx->Wm, ctx->Wb, ctx->Wq, ctx->G, ctx->partials,
                                                    ctx->n_partials, ctx->G_valid ? 1 : 0, ctx->n0,
                                                    ctx->colsq, c.renorm, c.nh, c.hd, c.hidden,
                                                    tpr);
  TTT_LAUNCH_CHECK(ctx, "commit_kernel");
  if (c.renorm) {
    int rc = launch_renorm_w2(ctx, nblk, s);
    if (rc != TTT_OK) return rc;
  }
  ctx->G_valid = false;
  ctx->n_partials = 0;
  return TTT_OK;
}

}  // namespace ttt
