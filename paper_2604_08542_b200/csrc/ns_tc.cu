// ns_tc.cu — Newton-Schulz orthonormalisation on the tensor cores (step 7 of the hot path; DESIGN.md
// reading R-NS; not in PAPER.md, required by BASELINE.json:north_star and configs 3 and 5).
//
// One CTA per gradient matrix X [H x hd] (hidden-major, tall: H >= hd). Tall form of the iteration:
//     X0 = g / (||g||_F + 1e-7),   g = (use_G ? G : 0) + sum_s P[s]      (fixed summation order)
//     n times:   A = X^T X  (hd x hd);   Pm = a I + b A + c A A;   X <- X Pm
// which is A = X X^T; X = a X + (b A + c A^2) X applied to g^T (NS(g^T) = NS(g)^T).
//
// Precision: a plain bf16 iteration misses the 2e-2 parity bar (the quintic amplifies operand
// rounding: slope a^5 ~ 485 at small singular values), so every product runs as a split-bf16
// ("bf16x3") contraction: each fp32 operand is held as hi + lo (two bf16), and the tensor cores
// accumulate hi*hi + hi*lo + lo*hi (+ lo*lo where it is free) in fp32 — about 16 mantissa bits per
// operand. Measured against the float64 oracle this keeps NS at the 5e-5 level.
//
// tcgen05 mapping (hd = 64; all operands in shared memory, 128-byte swizzle, fp32 accumulators in
// TMEM). X is kept as two bf16 tiles XH, XL [H rows][64], AL follows AH, XL follows XH, so that a
// 128-row operand is "hi stacked on lo":
//   Gram   D[128 x 64] = [XH | XL]^T (MN-major A, second 64-wide atom at LBO) . XH  then . XL
//          rows 0-63 = hi*hi + hi*lo, rows 64-127 = lo*hi + lo*lo;  A = top + bottom
//   square D[128 x 64] = [AH ; AL] (K-major A, 128 rows) . AH  then . AL;   A A = top + bottom
//   tall   D_mb[128 x 64] = XH_mb . PH + XH_mb . PL + XL_mb . PH        per 128-row block mb
// Phases are sequential (each product depends on the previous one): one elected thread issues the
// MMAs and commits to an mbarrier, all 8 warps run the TMEM -> registers -> split -> shared epilogue.
#include <stdio.h>

#include "tc_common.cuh"
#include "ttt_internal.h"

namespace ttt {

namespace nstc {
constexpr int THREADS = 256;
constexpr uint32_t C_A = 0;      // Gram accumulator        [128 x 64] fp32
constexpr uint32_t C_A2 = 64;    // A A accumulator         [128 x 64] fp32
constexpr uint32_t C_X = 128;    // X Pm accumulators, 64 columns per 128-row block
constexpr int S_LD = 65;         // fp32 exchange scratch row stride (bank-conflict free)
}  // namespace nstc

// hi/lo split of four fp32 values -> two 8-byte words of bf16
__device__ __forceinline__ void split4(const float (&v)[4], uint2& hi, uint2& lo) {
  hi.x = pack_bf16x2(v[0], v[1]);
  hi.y = pack_bf16x2(v[2], v[3]);
  float r[4];
  r[0] = v[0] - __uint_as_float(hi.x << 16);
  r[1] = v[1] - __uint_as_float(hi.x & 0xffff0000u);
  r[2] = v[2] - __uint_as_float(hi.y << 16);
  r[3] = v[3] - __uint_as_float(hi.y & 0xffff0000u);
  lo.x = pack_bf16x2(r[0], r[1]);
  lo.y = pack_bf16x2(r[2], r[3]);
}

// write 32 consecutive columns [c0, c0+32) of row `row` of a [rows][64] bf16 tile pair (hi, lo)
// in the 128-byte-swizzled layout (16-byte chunk index ^= row & 7)
__device__ __forceinline__ void store_row32_split(uint8_t* hi_tile, uint8_t* lo_tile, int row, int c0,
                                                  const float (&v)[32]) {
  const uint32_t swz = static_cast<uint32_t>(row & 7);
#pragma unroll
  for (int k = 0; k < 4; ++k) {            // 4 chunks of 8 columns
    const float a[4] = {v[8 * k], v[8 * k + 1], v[8 * k + 2], v[8 * k + 3]};
    const float b[4] = {v[8 * k + 4], v[8 * k + 5], v[8 * k + 6], v[8 * k + 7]};
    uint2 ha, la, hb, lb;
    split4(a, ha, la);
    split4(b, hb, lb);
    const uint32_t off = row * 128 + (((c0 >> 3) + k) ^ swz) * 16;
    *reinterpret_cast<uint4*>(hi_tile + off) = make_uint4(ha.x, ha.y, hb.x, hb.y);
    *reinterpret_cast<uint4*>(lo_tile + off) = make_uint4(la.x, la.y, lb.x, lb.y);
  }
}

__global__ void __launch_bounds__(nstc::THREADS, 1)
ns_tc_kernel(float* __restrict__ G, const float* __restrict__ P, int n_sets, size_t set_elems,
             int use_G, int H, int iters, uint32_t tmem_cols) {
  using namespace nstc;
  constexpr int HD = 64;
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) &
                                             ~static_cast<uintptr_t>(1023));
  __shared__ uint64_t mma_bar;
  __shared__ uint32_t tmem_base_s;
  __shared__ float red[THREADS / 32];
  __shared__ float s_scale;

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const uint32_t x_bytes = static_cast<uint32_t>(H) * 128u;
  uint8_t* XH = smem;
  uint8_t* XL = XH + x_bytes;
  uint8_t* AH = XL + x_bytes;
  uint8_t* AL = AH + 8192;
  uint8_t* PH = AL + 8192;
  uint8_t* PL = PH + 8192;
  float* S = reinterpret_cast<float*>(PL + 8192);          // [64][S_LD]

  if (tid == 0) { mbar_init(&mma_bar, 1); fence_mbar_init(); }
  if (warp == 0) { tmem_alloc(&tmem_base_s, tmem_cols); tmem_relinquish(); }

  // ---- load: g = (use_G ? G : 0) + sum_s P[s], written back to G; Frobenius norm ----
  const size_t mat_off = (size_t)blockIdx.x * H * HD;
  float* X = G + mat_off;
  const int n4 = H * HD / 4;
  float acc = 0.f;
  for (int e = tid; e < n4; e += THREADS) {
    float4 g = use_G ? reinterpret_cast<const float4*>(X)[e] : make_float4(0.f, 0.f, 0.f, 0.f);
    for (int s = 0; s < n_sets; ++s) {
      const float4 p = reinterpret_cast<const float4*>(P + (size_t)s * set_elems + mat_off)[e];
      g.x += p.x; g.y += p.y; g.z += p.z; g.w += p.w;
    }
    reinterpret_cast<float4*>(X)[e] = g;
    acc = fmaf(g.x, g.x, acc); acc = fmaf(g.y, g.y, acc);
    acc = fmaf(g.z, g.z, acc); acc = fmaf(g.w, g.w, acc);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  if (lane == 0) red[warp] = acc;
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tb = tmem_base_s;
  if (tid == 0) {
    float t = 0.f;
    for (int w = 0; w < THREADS / 32; ++w) t += red[w];
    s_scale = 1.0f / (sqrtf(t) + 1e-7f);
  }
  __syncthreads();
  const float scale = s_scale;
  for (int e = tid; e < n4; e += THREADS) {      // same thread re-reads what it wrote
    const float4 g = reinterpret_cast<const float4*>(X)[e];
    const float v[4] = {g.x * scale, g.y * scale, g.z * scale, g.w * scale};
    uint2 hi, lo;
    split4(v, hi, lo);
    const int row = e >> 4, c = (e & 15) * 4;    // 16 float4 per 64-wide row
    const uint32_t off = row * 128 + (((c >> 3) ^ (row & 7)) * 16) + (c & 7) * 2;
    *reinterpret_cast<uint2*>(XH + off) = hi;
    *reinterpret_cast<uint2*>(XL + off) = lo;
  }
  fence_proxy_async_smem();
  __syncthreads();

  constexpr uint32_t idesc_gram = umma_idesc_bf16(128, 64, 1, 1);   // A, B MN-major
  constexpr uint32_t idesc_kk = umma_idesc_bf16(128, 64, 0, 0);     // A, B K-major
  const uint32_t xh = smem_u32(XH), xl = smem_u32(XL), ah = smem_u32(AH), al = smem_u32(AL),
                 ph = smem_u32(PH), pl = smem_u32(PL);
  const int q = warp & 3, ch = warp >> 2;                     // TMEM lane quarter, column half
  const uint32_t lane_base = static_cast<uint32_t>(q * 32) << 16;
  const int c0 = 32 * ch;
  const int nblk = H / 128;
  const float ca = 3.4445f, cb = -4.7750f, cc = 2.0315f;
  uint32_t phase = 0;
  float Areg[32];

  // top (rows 0-63) + bottom (rows 64-127) of a [128 x 64] accumulator; result valid for q < 2
  auto fold_halves = [&](uint32_t col, float (&out)[32]) {
    uint32_t r[32];
    tmem_ld_x32(tb + lane_base + col + c0, r);
    tc_wait_ld();
    if (q >= 2) {
      float* dst = S + ((q - 2) * 32 + lane) * S_LD + c0;
#pragma unroll
      for (int j = 0; j < 32; ++j) dst[j] = __uint_as_float(r[j]);
    }
    __syncthreads();
    if (q < 2) {
      const float* src = S + (q * 32 + lane) * S_LD + c0;
#pragma unroll
      for (int j = 0; j < 32; ++j) out[j] = __uint_as_float(r[j]) + src[j];
    }
  };
  auto end_phase = [&]() {
    fence_proxy_async_smem();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
  };
  auto wait_mma = [&]() {
    mbar_wait(&mma_bar, phase & 1);
    phase ^= 1;
    tc_fence_after();
  };

  for (int it = 0; it < iters; ++it) {
    // ---------------- A = X^T X ----------------
    if (tid == 0) {
      for (int ks = 0; ks < H / 16; ++ks) {
        const uint64_t a = umma_smem_desc_sw128(xh + 2048 * ks, x_bytes, 1024);
        umma_ss(tb + C_A, a, umma_smem_desc_sw128(xh + 2048 * ks, x_bytes, 1024), idesc_gram, ks > 0);
        umma_ss(tb + C_A, a, umma_smem_desc_sw128(xl + 2048 * ks, x_bytes, 1024), idesc_gram, 1);
      }
      tc_commit(&mma_bar);
    }
    wait_mma();
    fold_halves(C_A, Areg);
    if (q < 2) store_row32_split(AH, AL, q * 32 + lane, c0, Areg);
    end_phase();
    // ---------------- Pm = a I + b A + c A A ----------------
    if (tid == 0) {
#pragma unroll
      for (int k = 0; k < HD / 16; ++k) {
        const uint64_t a = umma_smem_desc_sw128(ah + 32 * k, 16, 1024);   // 128 rows: AH then AL
        umma_ss(tb + C_A2, a, umma_smem_desc_sw128(ah + 32 * k, 16, 1024), idesc_kk, k > 0);
        umma_ss(tb + C_A2, a, umma_smem_desc_sw128(al + 32 * k, 16, 1024), idesc_kk, 1);
      }
      tc_commit(&mma_bar);
    }
    wait_mma();
    {
      float A2[32];
      fold_halves(C_A2, A2);
      if (q < 2) {
        const int row = q * 32 + lane;
#pragma unroll
        for (int j = 0; j < 32; ++j) {
          float p = fmaf(cc, A2[j], cb * Areg[j]);
          if (c0 + j == row) p += ca;
          A2[j] = p;
        }
        store_row32_split(PH, PL, row, c0, A2);
      }
    }
    end_phase();
    // ---------------- X <- X Pm ----------------
    if (tid == 0) {
      for (int mb = 0; mb < nblk; ++mb) {
        const uint32_t d = tb + C_X + 64 * mb;
        const uint32_t xhb = xh + mb * (128 * 128), xlb = xl + mb * (128 * 128);
#pragma unroll
        for (int k = 0; k < HD / 16; ++k) {
          const uint64_t a_hi = umma_smem_desc_sw128(xhb + 32 * k, 16, 1024);
          const uint64_t b_hi = umma_smem_desc_sw128(ph + 32 * k, 16, 1024);
          umma_ss(d, a_hi, b_hi, idesc_kk, k > 0);
          umma_ss(d, a_hi, umma_smem_desc_sw128(pl + 32 * k, 16, 1024), idesc_kk, 1);
          umma_ss(d, umma_smem_desc_sw128(xlb + 32 * k, 16, 1024), b_hi, idesc_kk, 1);
        }
      }
      tc_commit(&mma_bar);
    }
    wait_mma();
    for (int mb = 0; mb < nblk; ++mb) {
      uint32_t r[32];
      tmem_ld_x32(tb + lane_base + C_X + 64 * mb + c0, r);
      tc_wait_ld();
      const int row = mb * 128 + q * 32 + lane;
      if (it == iters - 1) {
        float4* dst = reinterpret_cast<float4*>(X + (size_t)row * HD + c0);
#pragma unroll
        for (int v = 0; v < 8; ++v)
          dst[v] = make_float4(__uint_as_float(r[4 * v]), __uint_as_float(r[4 * v + 1]),
                               __uint_as_float(r[4 * v + 2]), __uint_as_float(r[4 * v + 3]));
      } else {
        float f[32];
#pragma unroll
        for (int j = 0; j < 32; ++j) f[j] = __uint_as_float(r[j]);
        store_row32_split(XH, XL, row, c0, f);
      }
    }
    end_phase();
  }
  if (warp == 0) tmem_dealloc(tb, tmem_cols);
}

int ns_tc_supported(const ttt_config* cfg) {
  return cfg->act_dtype == TTT_BF16 && cfg->hd == 64 && cfg->hidden % 128 == 0 &&
         cfg->hidden >= 128 && cfg->hidden <= 512 && !cfg->linear_fast_weight;
}

// In-place NS of all 3*nh matrices of the pending gradient; folds the partial sets into G first.
int launch_ns_tc(ttt_ctx* ctx, cudaStream_t s) {
  const ttt_config& c = ctx->cfg;
  const size_t smem = (size_t)2 * c.hidden * 128 + 4 * 8192 + 64 * nstc::S_LD * sizeof(float) + 1024;
  static size_t attr_smem = 0;
  if (smem > attr_smem) {
    TTT_CUDA_TRY(ctx, cudaFuncSetAttribute(ns_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                           (int)smem), "ns_tc_kernel smem attr");
    attr_smem = smem;
  }
  uint32_t cols = 128 + 64 * (c.hidden / 128);
  uint32_t alloc = 32;
  while (alloc < cols) alloc <<= 1;
  ns_tc_kernel<<<3 * c.nh, nstc::THREADS, smem, s>>>(ctx->G, ctx->partials, ctx->n_partials,
                                                     3 * ctx->mat_elems, ctx->G_valid ? 1 : 0,
                                                     c.hidden, c.ns_iters, alloc);
  TTT_LAUNCH_CHECK(ctx, "ns_tc_kernel");
  ctx->G_valid = true;
  ctx->n_partials = 0;
  return TTT_OK;
}

}  // namespace ttt
