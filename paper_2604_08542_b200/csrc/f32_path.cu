// f32_path.cu — the fp32 path (cfg.act_dtype == TTT_F32): every contraction in fp32 FFMA on the
// CUDA cores (single-pass TF32 would miss the 1e-4 bar of BASELINE.json:north_star). It serves the
// tiny parity configuration (BASELINE.json:configs[0]) and the linear closed-form test mode; it
// is not a performance path, so the hidden activations round-trip through an fp32 workspace.
//
//   accumulate:  fwd kernel   A = K W1, B = K W3, g = V W2^T            (Eq. 12, steps 1 and 3)
//                             Hd' = -eta Hd, dA, dB                      (SwiGLU fwd/bwd epilogue)
//                grad kernel  G1^T = dA^T K, G3^T = dB^T K, G2 = Hd'^T V (Eq. 8) -> partial sets
//   apply:       fwd kernel   Hq = SiLU(Q W1) o (Q W3);  out kernel  O = Hq W2         (Eq. 4)
#include "ttt_internal.h"

namespace ttt {

constexpr int TS = 64;   // output tile 64 x 64
constexpr int TK = 16;   // contraction step
constexpr int F32_THREADS = 256;

// acc[4][4] += sum_{k in [0,kdim)} A(m0+4ty+r, k) * B(k, n0+4tx+c)
// A(m,k) at A[m*a_rs + k*a_cs], valid for m < mmax; B(k,n) at B[k*b_rs + n*b_cs], n < nmax.
__device__ __forceinline__ void simt_gemm_tile(const float* __restrict__ A, long a_rs, long a_cs,
                                               int m0, int mmax, const float* __restrict__ B,
                                               long b_rs, long b_cs, int n0, int nmax, int kdim,
                                               float (&acc)[4][4], float (*As)[TS + 4],
                                               float (*Bs)[TS + 4]) {
  const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
  for (int k0 = 0; k0 < kdim; k0 += TK) {
    __syncthreads();
#pragma unroll
    for (int l = 0; l < (TS * TK) / F32_THREADS; ++l) {
      const int e = tid + l * F32_THREADS;
      int m, k;
      if (a_cs == 1) { m = e / TK; k = e % TK; } else { k = e / TS; m = e % TS; }
      const bool ok = (m0 + m < mmax) && (k0 + k < kdim);
      As[k][m] = ok ? A[(long)(m0 + m) * a_rs + (long)(k0 + k) * a_cs] : 0.f;
      int n, kb;
      if (b_rs == 1) { n = e / TK; kb = e % TK; } else { kb = e / TS; n = e % TS; }
      const bool okb = (n0 + n < nmax) && (k0 + kb < kdim);
      Bs[kb][n] = okb ? B[(long)(k0 + kb) * b_rs + (long)(n0 + n) * b_cs] : 0.f;
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < TK; ++k) {
      float a[4], b[4];
#pragma unroll
      for (int r = 0; r < 4; ++r) a[r] = As[k][ty * 4 + r];
#pragma unroll
      for (int c = 0; c < 4; ++c) b[c] = Bs[k][tx * 4 + c];
#pragma unroll
      for (int r = 0; r < 4; ++r)
#pragma unroll
        for (int c = 0; c < 4; ++c) acc[r][c] = fmaf(a[r], b[c], acc[r][c]);
    }
  }
}

__device__ __forceinline__ float sigmoid_f32(float a) {
  // accurate form: fp32 path is held to 1e-4 against the float64 oracle
  return a >= 0.f ? 1.f / (1.f + expf(-a)) : expf(a) / (1.f + expf(a));
}

// MODE 0: update forward + SwiGLU backward epilogue; X = K, Y = V. Writes act0 = dA, act1 = dB,
//         act2 = Hd' = -eta*Hd  ([nh][M][H]) and per-block loss partials.
// MODE 1: apply forward; X = Q. Writes act0 = Hq.
// MODE 2: linear test mode update: act0 = -eta*V (H == hd), loss = sum (K W1) o (-eta V).
// MODE 3: linear test mode apply: O = X W1 written to Out directly (H == hd).
// grid (ceil(H/64), ceil(M/64), nh)
template <int MODE>
__global__ void __launch_bounds__(F32_THREADS)
f32_fwd_kernel(const float* __restrict__ X, const float* __restrict__ Y, const float* __restrict__ lr,
               const float* __restrict__ Wm, float* __restrict__ act0, float* __restrict__ act1,
               float* __restrict__ act2, float* __restrict__ Out, float* __restrict__ loss_blk,
               int M, long ld, int nh, int hd, int H) {
  __shared__ float As[TK][TS + 4];
  __shared__ float Bs[TK][TS + 4];
  __shared__ float red[F32_THREADS / 32];
  const int h = blockIdx.z, t0 = blockIdx.y * TS, j0 = blockIdx.x * TS;
  const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
  const size_t me = (size_t)nh * H * hd;
  const float* W1t = Wm + (size_t)h * H * hd;           // [H][hd]
  const float* W2 = Wm + me + (size_t)h * H * hd;       // [H][hd]
  const float* W3t = Wm + 2 * me + (size_t)h * H * hd;  // [H][hd]
  const float* Xh = X + (size_t)h * hd;

  float a[4][4] = {}, b[4][4] = {}, g[4][4] = {};
  // A[t][j] = sum_i X[t][i] W1t[j][i]
  simt_gemm_tile(Xh, ld, 1, t0, M, W1t, 1, hd, j0, H, hd, a, As, Bs);
  if (MODE == 0 || MODE == 1) simt_gemm_tile(Xh, ld, 1, t0, M, W3t, 1, hd, j0, H, hd, b, As, Bs);
  if (MODE == 0) simt_gemm_tile(Y + (size_t)h * hd, ld, 1, t0, M, W2, 1, hd, j0, H, hd, g, As, Bs);

  float loss = 0.f;
#pragma unroll
  for (int r = 0; r < 4; ++r) {
    const int t = t0 + ty * 4 + r;
    if (t >= M) continue;
    const float ne = (MODE == 0 || MODE == 2) ? -lr[(size_t)h * M + t] : 0.f;
#pragma unroll
    for (int c = 0; c < 4; ++c) {
      const int j = j0 + tx * 4 + c;
      if (j >= H) continue;
      const size_t o = ((size_t)h * M + t) * H + j;
      if (MODE == 0) {
        const float av = a[r][c], bv = b[r][c];
        const float s = sigmoid_f32(av);
        const float S = av * s;                 // SiLU(a)
        const float hdv = S * bv;               // hidden activation
        const float dhd = ne * g[r][c];         // dHd = (-eta v) W2^T
        act0[o] = dhd * bv * (s * (1.f + av * (1.f - s)));  // dA
        act1[o] = dhd * S;                                   // dB
        act2[o] = ne * hdv;                                  // Hd' (for G2 = Hd'^T V)
        loss = fmaf(hdv, dhd, loss);
      } else if (MODE == 1) {
        const float av = a[r][c];
        act0[o] = av * sigmoid_f32(av) * b[r][c];
      } else if (MODE == 2) {
        const float dy = ne * Y[(size_t)t * ld + (size_t)h * hd + j];
        act0[o] = dy;
        loss = fmaf(a[r][c], dy, loss);
      } else {
        Out[(size_t)t * ld + (size_t)h * hd + j] = a[r][c];
      }
    }
  }
  if (MODE == 0 || MODE == 2) {
    if (loss_blk != nullptr) {
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) loss += __shfl_xor_sync(0xffffffffu, loss, o);
      if ((tid & 31) == 0) red[tid >> 5] = loss;
      __syncthreads();
      if (tid == 0) {
        float t = 0.f;
        for (int w = 0; w < F32_THREADS / 32; ++w) t += red[w];
        loss_blk[((size_t)h * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x] = t;
      }
    }
  }
}

// loss_part[split][h] = sum over the fwd blocks of this split's token range, fixed order
__global__ void f32_loss_split_kernel(const float* __restrict__ loss_blk, float* __restrict__ part,
                                      int nh, int ny, int nx, int tiles_per_split) {
  const int h = blockIdx.x, sp = blockIdx.y;
  if (threadIdx.x != 0) return;
  float t = 0.f;
  const int y0 = sp * tiles_per_split, y1 = min(ny, y0 + tiles_per_split);
  for (int y = y0; y < y1; ++y)
    for (int x = 0; x < nx; ++x) t += loss_blk[((size_t)h * ny + y) * nx + x];
  part[(size_t)sp * nh + h] = t;
}

// partial gradients over one token range: P[split][mat][h][j][i] = sum_t act_mat[h][t][j] * Y_mat[t][i]
// mat 0: dA^T K, mat 1: Hd'^T V, mat 2: dB^T K.  grid (ceil(H/64)*ceil(hd/64), nh*3, splits)
__global__ void __launch_bounds__(F32_THREADS)
f32_grad_kernel(const float* __restrict__ K, const float* __restrict__ V,
                const float* __restrict__ act0, const float* __restrict__ act1,
                const float* __restrict__ act2, float* __restrict__ P, int M, long ld, int nh,
                int hd, int H, int tokens_per_split, int linear) {
  __shared__ float As[TK][TS + 4];
  __shared__ float Bs[TK][TS + 4];
  const int ni = (hd + TS - 1) / TS;
  const int j0 = (blockIdx.x / ni) * TS, i0 = (blockIdx.x % ni) * TS;
  const int mat = blockIdx.y % 3, h = blockIdx.y / 3, sp = blockIdx.z;
  const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
  const int tlo = sp * tokens_per_split, thi = min(M, tlo + tokens_per_split);
  const float* act = (mat == 0 ? act0 : mat == 1 ? act2 : act1) + ((size_t)h * M + tlo) * H;
  const float* Y = (mat == 1 ? V : K) + (size_t)tlo * ld + (size_t)h * hd;
  float acc[4][4] = {};
  // out[j][i] = sum_t act[t][j] * Y[t][i]:  A(m=j,k=t) at act[t*H + j], B(k=t,n=i) at Y[t*ld + i]
  if (!(linear && mat != 0) && thi > tlo)
    simt_gemm_tile(act, 1, H, j0, H, Y, ld, 1, i0, hd, thi - tlo, acc, As, Bs);
  const size_t me = (size_t)nh * H * hd;
  float* out = P + (size_t)sp * 3 * me + mat * me + (size_t)h * H * hd;
#pragma unroll
  for (int r = 0; r < 4; ++r) {
    const int j = j0 + ty * 4 + r;
    if (j >= H) continue;
#pragma unroll
    for (int c = 0; c < 4; ++c) {
      const int i = i0 + tx * 4 + c;
      if (i < hd) out[(size_t)j * hd + i] = acc[r][c];
    }
  }
}

// O[t][i] = sum_j Hq[h][t][j] * W2[j][i].  grid (ceil(hd/64), ceil(M/64), nh)
__global__ void __launch_bounds__(F32_THREADS)
f32_out_kernel(const float* __restrict__ Hq, const float* __restrict__ Wm, float* __restrict__ O,
               int M, long ld, int nh, int hd, int H) {
  __shared__ float As[TK][TS + 4];
  __shared__ float Bs[TK][TS + 4];
  const int h = blockIdx.z, t0 = blockIdx.y * TS, i0 = blockIdx.x * TS;
  const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
  const size_t me = (size_t)nh * H * hd;
  const float* W2 = Wm + me + (size_t)h * H * hd;
  float acc[4][4] = {};
  simt_gemm_tile(Hq + (size_t)h * M * H, H, 1, t0, M, W2, hd, 1, i0, hd, H, acc, As, Bs);
#pragma unroll
  for (int r = 0; r < 4; ++r) {
    const int t = t0 + ty * 4 + r;
    if (t >= M) continue;
#pragma unroll
    for (int c = 0; c < 4; ++c) {
      const int i = i0 + tx * 4 + c;
      if (i < hd) O[(size_t)t * ld + (size_t)h * hd + i] = acc[r][c];
    }
  }
}

// bf16 <-> fp32 conversion of token tensors (bf16 I/O on this path): 8 elements per thread
__global__ void bf16_to_f32_kernel(const __nv_bfloat16* __restrict__ src, long ld, float* __restrict__ dst,
                                   long M, int cols) {
  const long e = ((long)blockIdx.x * blockDim.x + threadIdx.x) * 8;
  if (e >= M * cols) return;
  const long r = e / cols, c = e % cols;
  const uint4 x = *reinterpret_cast<const uint4*>(src + r * ld + c);
  const uint32_t w[4] = {x.x, x.y, x.z, x.w};
  float4 a, b;
  a.x = __uint_as_float(w[0] << 16); a.y = __uint_as_float(w[0] & 0xffff0000u);
  a.z = __uint_as_float(w[1] << 16); a.w = __uint_as_float(w[1] & 0xffff0000u);
  b.x = __uint_as_float(w[2] << 16); b.y = __uint_as_float(w[2] & 0xffff0000u);
  b.z = __uint_as_float(w[3] << 16); b.w = __uint_as_float(w[3] & 0xffff0000u);
  reinterpret_cast<float4*>(dst + e)[0] = a;
  reinterpret_cast<float4*>(dst + e)[1] = b;
}
__global__ void f32_to_bf16_kernel(const float* __restrict__ src, __nv_bfloat16* __restrict__ dst, long ld,
                                   long M, int cols) {
  const long e = ((long)blockIdx.x * blockDim.x + threadIdx.x) * 8;
  if (e >= M * cols) return;
  const long r = e / cols, c = e % cols;
  const float4 a = reinterpret_cast<const float4*>(src + e)[0], b = reinterpret_cast<const float4*>(src + e)[1];
  __nv_bfloat162 p0 = __floats2bfloat162_rn(a.x, a.y), p1 = __floats2bfloat162_rn(a.z, a.w),
                 p2 = __floats2bfloat162_rn(b.x, b.y), p3 = __floats2bfloat162_rn(b.z, b.w);
  uint4 o;
  o.x = *reinterpret_cast<uint32_t*>(&p0); o.y = *reinterpret_cast<uint32_t*>(&p1);
  o.z = *reinterpret_cast<uint32_t*>(&p2); o.w = *reinterpret_cast<uint32_t*>(&p3);
  *reinterpret_cast<uint4*>(dst + r * ld + c) = o;
}

int launch_bf16_to_f32(ttt_ctx* ctx, const __nv_bfloat16* src, int64_t ld, float* dst, int64_t M, cudaStream_t s) {
  const int cols = ctx->cfg.nh * ctx->cfg.hd;
  const long n8 = (long)M * cols / 8;
  bf16_to_f32_kernel<<<(unsigned)((n8 + 255) / 256), 256, 0, s>>>(src, ld, dst, M, cols);
  TTT_LAUNCH_CHECK(ctx, "bf16_to_f32_kernel");
  return TTT_OK;
}
int launch_f32_to_bf16(ttt_ctx* ctx, const float* src, __nv_bfloat16* dst, int64_t ld, int64_t M, cudaStream_t s) {
  const int cols = ctx->cfg.nh * ctx->cfg.hd;
  const long n8 = (long)M * cols / 8;
  f32_to_bf16_kernel<<<(unsigned)((n8 + 255) / 256), 256, 0, s>>>(src, dst, ld, M, cols);
  TTT_LAUNCH_CHECK(ctx, "f32_to_bf16_kernel");
  return TTT_OK;
}

// ------------------------------------------------------------------------------------------------
static int f32_splits(const ttt_ctx* ctx, int64_t M, int* tokens_per_split) {
  // token ranges are multiples of the 64-token fwd tile so loss partials map onto splits
  const int64_t tiles = (M + TS - 1) / TS;
  int64_t want = (ctx->sm_count * 2) / (3 * ctx->cfg.nh * ((ctx->cfg.hidden + TS - 1) / TS)) + 1;
  if (want > tiles) want = tiles;
  if (want > 16) want = 16;
  if (want < 1) want = 1;
  const int64_t tps = (tiles + want - 1) / want;
  *tokens_per_split = (int)(tps * TS);
  return (int)((tiles + tps - 1) / tps);
}

int f32_partials_needed(const ttt_ctx* ctx, int64_t M) {
  int tps;
  return f32_splits(ctx, M, &tps);
}

int f32_accumulate(ttt_ctx* ctx, const float* K, const float* V, const float* lr, int64_t M,
                   int64_t ld, bool want_loss, int* used, int* loss_rows, cudaStream_t s) {
  const ttt_config& c = ctx->cfg;
  const int H = c.hidden, hd = c.hd, nh = c.nh;
  int tps;
  const int splits = f32_splits(ctx, M, &tps);
  dim3 gf((H + TS - 1) / TS, (unsigned)((M + TS - 1) / TS), nh);
  float* loss_blk = want_loss ? ctx->loss_blk : nullptr;
  if (c.linear_fast_weight) {
    f32_fwd_kernel<2><<<gf, F32_THREADS, 0, s>>>(K, V, lr, ctx->Wm, ctx->act[0], nullptr, nullptr,
                                                 nullptr, loss_blk, (int)M, ld, nh, hd, H);
  } else {
    f32_fwd_kernel<0><<<gf, F32_THREADS, 0, s>>>(K, V, lr, ctx->Wm, ctx->act[0], ctx->act[1],
                                                 ctx->act[2], nullptr, loss_blk, (int)M, ld, nh,
                                                 hd, H);
  }
  TTT_LAUNCH_CHECK(ctx, "f32_fwd_kernel");
  float* P = ctx->partials + (size_t)ctx->n_partials * 3 * ctx->mat_elems;
  dim3 gg(((H + TS - 1) / TS) * ((hd + TS - 1) / TS), nh * 3, splits);
  f32_grad_kernel<<<gg, F32_THREADS, 0, s>>>(K, V, ctx->act[0], ctx->act[1], ctx->act[2], P, (int)M,
                                             ld, nh, hd, H, tps, c.linear_fast_weight);
  TTT_LAUNCH_CHECK(ctx, "f32_grad_kernel");
  if (want_loss) {
    f32_loss_split_kernel<<<dim3(nh, splits), 32, 0, s>>>(
        loss_blk, ctx->loss_part, nh, gf.y, gf.x, tps / TS);
    TTT_LAUNCH_CHECK(ctx, "f32_loss_split_kernel");
  }
  *used = splits;
  *loss_rows = splits;
  return TTT_OK;
}

int f32_apply(ttt_ctx* ctx, const float* Q, float* O, int64_t M, int64_t ld, cudaStream_t s) {
  const ttt_config& c = ctx->cfg;
  const int H = c.hidden, hd = c.hd, nh = c.nh;
  dim3 gf((H + TS - 1) / TS, (unsigned)((M + TS - 1) / TS), nh);
  if (c.linear_fast_weight) {
    f32_fwd_kernel<3><<<gf, F32_THREADS, 0, s>>>(Q, nullptr, nullptr, ctx->Wm, nullptr, nullptr,
                                                 nullptr, O, nullptr, (int)M, ld, nh, hd, H);
    TTT_LAUNCH_CHECK(ctx, "f32_fwd_kernel<3>");
    return TTT_OK;
  }
  f32_fwd_kernel<1><<<gf, F32_THREADS, 0, s>>>(Q, nullptr, nullptr, ctx->Wm, ctx->act[0], nullptr,
                                               nullptr, nullptr, nullptr, (int)M, ld, nh, hd, H);
  TTT_LAUNCH_CHECK(ctx, "f32_fwd_kernel<1>");
  dim3 go((hd + TS - 1) / TS, (unsigned)((M + TS - 1) / TS), nh);
  f32_out_kernel<<<go, F32_THREADS, 0, s>>>(ctx->act[0], ctx->Wm, O, (int)M, ld, nh, hd, H);
  TTT_LAUNCH_CHECK(ctx, "f32_out_kernel");
  return TTT_OK;
}

}  // namespace ttt
