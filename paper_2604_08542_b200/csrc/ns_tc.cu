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
//   Gram   D[128 x 128] = [XH | XL]^T . [XH | XL]   (MN-major A and B, second 64-wide atom at LBO)
//          four 64 x 64 blocks hh, hl / lh, ll in ONE MMA per 16 rows;  A = sum of the four blocks
//   square D[128 x 128] = [AH ; AL] . [AH ; AL]^T  (K-major, 128 rows each);  A A = sum of the blocks
//   tall   D_mb[128 x 128] = XH_mb . [PH ; PL]^T, then columns 0-63 += XL_mb . PH^T   per 128-row block
//          X' = left half + right half
// SS-mode MMAs with a 64-wide dimension are bound by the shared-memory operand port (128 B/clk),
// which is why the hi/lo halves are stacked into 128-wide operands instead of issued as three
// 64-wide products. Phases are sequential (each product depends on the previous one): one elected
// thread of a dedicated warp issues the MMAs and commits to an mbarrier, 16 worker warps run the
// TMEM -> registers -> split -> shared epilogue (4 warps per TMEM lane quarter, 16 columns each).
#include <stdio.h>

#include "tc_common.cuh"
#include "ttt_internal.h"

namespace ttt {

namespace nstc {
constexpr int THREADS = 512;     // epilogue / load workers (16 warps)
constexpr int LAUNCH_THREADS = THREADS + 32;   // + a dedicated MMA-issuing warp (warp 16)
constexpr uint32_t C_A = 0;      // Gram accumulator   [128 x 128] fp32
constexpr uint32_t C_A2 = 128;   // A A accumulator    [128 x 128] fp32
constexpr uint32_t C_X = 0;      // X Pm accumulators, 128 columns per 128-row block (alias C_A, C_A2)
constexpr int S_LD = 65;         // fp32 exchange scratch row stride in floats (bank-conflict free)
constexpr int W_LD = 68;         // fp32 commit staging row stride in floats (16-B aligned rows)
}  // namespace nstc

// hi/lo split of eight fp32 values -> one 16-byte chunk of bf16 each
__device__ __forceinline__ void split8(const float (&v)[8], uint4& hi, uint4& lo) {
  uint32_t h[4], l[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    h[i] = pack_bf16x2(v[2 * i], v[2 * i + 1]);
    const float r0 = v[2 * i] - __uint_as_float(h[i] << 16);
    const float r1 = v[2 * i + 1] - __uint_as_float(h[i] & 0xffff0000u);
    l[i] = pack_bf16x2(r0, r1);
  }
  hi = make_uint4(h[0], h[1], h[2], h[3]);
  lo = make_uint4(l[0], l[1], l[2], l[3]);
}

// byte offset of 16-byte chunk `chunk` (8 bf16 columns) of row `row` in a 128-byte-swizzled
// [rows][64] bf16 tile
__device__ __forceinline__ uint32_t sw128_off(int row, int chunk) {
  return static_cast<uint32_t>(row * 128 + ((chunk ^ (row & 7)) << 4));
}

__global__ void __launch_bounds__(nstc::LAUNCH_THREADS, 1)
ns_tc_kernel(float* __restrict__ G, const float* __restrict__ P, int n_sets, size_t set_elems,
             int use_G, int H, int iters, uint32_t tmem_cols, float* __restrict__ Wm,
             ttt_wop_t* __restrict__ Wb) {
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
  const bool issuer = warp == THREADS / 32;    // issues every MMA; takes part in the CTA barriers only
  const uint32_t x_bytes = static_cast<uint32_t>(H) * 128u;
  uint8_t* XH = smem;
  uint8_t* XL = XH + x_bytes;
  uint8_t* AH = XL + x_bytes;
  uint8_t* AL = AH + 8192;
  uint8_t* PH = AL + 8192;
  uint8_t* PL = PH + 8192;
  float* S = reinterpret_cast<float*>(PL + 8192);          // [128][S_LD]

  if (tid == 0) { mbar_init(&mma_bar, 1); fence_mbar_init(); }
  if (warp == 0) { tmem_alloc(&tmem_base_s, tmem_cols); tmem_relinquish(); }
  // programmatic dependent launch: the set-up above overlapped the tail of the gradient kernel
  asm volatile("griddepcontrol.wait;" ::: "memory");

  // ---- load: g = (use_G ? G : 0) + sum_s P[s] (fixed order), written back to G; Frobenius norm ----
  const size_t mat_off = (size_t)blockIdx.x * H * HD;
  float* X = G + mat_off;
  const int n4 = H * HD / 4;
  constexpr int LB = 4;                            // float4 loads in flight per thread and set
  float acc = 0.f;
  for (int e0 = issuer ? n4 : tid; e0 < n4; e0 += THREADS * LB) {
    float4 g[LB];
#pragma unroll
    for (int u = 0; u < LB; ++u) {
      const int e = e0 + u * THREADS;
      g[u] = (use_G && e < n4) ? reinterpret_cast<const float4*>(X)[e] : make_float4(0.f, 0.f, 0.f, 0.f);
    }
    for (int s0 = 0; s0 < n_sets; s0 += 4) {       // 4 sets x LB loads in flight, summed in set order
      float4 p[4][LB];
#pragma unroll
      for (int ds = 0; ds < 4; ++ds) {
        const float4* ps = reinterpret_cast<const float4*>(P + (size_t)(s0 + ds) * set_elems + mat_off);
#pragma unroll
        for (int u = 0; u < LB; ++u) {
          const int e = e0 + u * THREADS;
          p[ds][u] = (s0 + ds < n_sets && e < n4) ? __ldcg(ps + e) : make_float4(0.f, 0.f, 0.f, 0.f);
        }
      }
#pragma unroll
      for (int ds = 0; ds < 4; ++ds)
#pragma unroll
        for (int u = 0; u < LB; ++u) {
          g[u].x += p[ds][u].x; g[u].y += p[ds][u].y; g[u].z += p[ds][u].z; g[u].w += p[ds][u].w;
        }
    }
#pragma unroll
    for (int u = 0; u < LB; ++u) {
      const int e = e0 + u * THREADS;
      if (e < n4) {
        reinterpret_cast<float4*>(X)[e] = g[u];
        acc = fmaf(g[u].x, g[u].x, acc); acc = fmaf(g[u].y, g[u].y, acc);
        acc = fmaf(g[u].z, g[u].z, acc); acc = fmaf(g[u].w, g[u].w, acc);
      }
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  if (lane == 0 && !issuer) red[warp] = acc;
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
  for (int e0 = issuer ? n4 : tid; e0 < n4; e0 += THREADS * LB) {   // same thread re-reads what it wrote
    float4 g[LB];
#pragma unroll
    for (int u = 0; u < LB; ++u) {
      const int e = e0 + u * THREADS;
      g[u] = e < n4 ? reinterpret_cast<const float4*>(X)[e] : make_float4(0.f, 0.f, 0.f, 0.f);
    }
#pragma unroll
    for (int u = 0; u < LB; ++u) {
      const int e = e0 + u * THREADS;
      if (e < n4) {
        const float v0 = g[u].x * scale, v1 = g[u].y * scale, v2 = g[u].z * scale, v3 = g[u].w * scale;
        uint2 hi, lo;
        hi.x = pack_bf16x2(v0, v1);
        hi.y = pack_bf16x2(v2, v3);
        lo.x = pack_bf16x2(v0 - __uint_as_float(hi.x << 16), v1 - __uint_as_float(hi.x & 0xffff0000u));
        lo.y = pack_bf16x2(v2 - __uint_as_float(hi.y << 16), v3 - __uint_as_float(hi.y & 0xffff0000u));
        const int row = e >> 4, c = (e & 15) * 4;    // 16 float4 per 64-wide row
        const uint32_t off = sw128_off(row, c >> 3) + (c & 7) * 2;
        *reinterpret_cast<uint2*>(XH + off) = hi;
        *reinterpret_cast<uint2*>(XL + off) = lo;
      }
    }
  }
  fence_proxy_async_smem();
  __syncthreads();

  constexpr uint32_t idesc_gram = umma_idesc_bf16(128, 128, 1, 1);  // A, B MN-major, hi | lo atoms
  constexpr uint32_t idesc_k128 = umma_idesc_bf16(128, 128, 0, 0);  // A, B K-major, 128 rows each
  constexpr uint32_t idesc_k64 = umma_idesc_bf16(128, 64, 0, 0);
  // shared-memory matrix descriptors; an address step of b bytes is +(b >> 4) on the descriptor
  const uint64_t d_x_mn = umma_smem_desc_sw128(smem_u32(XH), x_bytes, 1024);    // MN-major, 2nd atom = XL
  const uint64_t d_xh_k = umma_smem_desc_sw128(smem_u32(XH), 16, 1024);         // K-major
  const uint64_t d_xl_k = umma_smem_desc_sw128(smem_u32(XL), 16, 1024);
  const uint64_t d_a = umma_smem_desc_sw128(smem_u32(AH), 16, 1024);            // 128 rows: AH then AL
  const uint64_t d_p = umma_smem_desc_sw128(smem_u32(PH), 16, 1024);            // 128 rows: PH then PL
  const int q = warp & 3, cs = warp >> 2;                     // TMEM lane quarter, 16-column group
  const uint32_t lane_base = static_cast<uint32_t>(q * 32) << 16;
  const int trow = q * 32 + lane;                             // accumulator row this thread reads
  const int frow = tid & 63, fch = tid >> 6;                  // fold mapping: row, 8-column chunk
  const int nblk = H / 128;
  const float ca = 3.4445f, cb = -4.7750f, cc = 2.0315f;
  uint32_t phase = 0;
  float Areg[8];

  // sum of the four 64 x 64 blocks of a [128 x 128] accumulator -> 8 values (frow, 8 fch + j):
  // part 1 (workers) column halves added, rows exported; CTA barrier; part 2 top + bottom rows
  auto fold_export = [&](uint32_t col) {
    uint32_t r0[16], r1[16];
    tmem_ld_x16(tb + lane_base + col + 16 * cs, r0);
    tmem_ld_x16(tb + lane_base + col + 64 + 16 * cs, r1);
    tc_wait_ld();
    float* dst = S + trow * S_LD + 16 * cs;
#pragma unroll
    for (int j = 0; j < 16; ++j) dst[j] = __uint_as_float(r0[j]) + __uint_as_float(r1[j]);
  };
  auto fold_import = [&](float (&out)[8]) {
    const float* top = S + frow * S_LD + 8 * fch;
    const float* bot = top + 64 * S_LD;
#pragma unroll
    for (int j = 0; j < 8; ++j) out[j] = top[j] + bot[j];
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
  const uint32_t lead = issuer ? elect_one() : 0u;

  for (int it = 0; it < iters; ++it) {
    const bool last = it == iters - 1;
    // ---------------- A = X^T X ----------------
    if (lead) {
      uint64_t d = d_x_mn;                                  // +2048 B per 16-row K step
      for (int ks = 0; ks < H / 16; ++ks, d += 128) umma_ss(tb + C_A, d, d, idesc_gram, ks > 0);
      tc_commit(&mma_bar);
    }
    if (!issuer) { wait_mma(); fold_export(C_A); }
    __syncthreads();
    if (!issuer) {
      fold_import(Areg);
      uint4 hi, lo;
      split8(Areg, hi, lo);
      *reinterpret_cast<uint4*>(AH + sw128_off(frow, fch)) = hi;
      *reinterpret_cast<uint4*>(AL + sw128_off(frow, fch)) = lo;
    }
    end_phase();
    // ---------------- Pm = a I + b A + c A A ----------------
    if (lead) {
#pragma unroll
      for (int k = 0; k < HD / 16; ++k)                     // +32 B per 16-column K step
        umma_ss(tb + C_A2, d_a + 2 * k, d_a + 2 * k, idesc_k128, k > 0);
      tc_commit(&mma_bar);
    }
    if (!issuer) { wait_mma(); fold_export(C_A2); }
    __syncthreads();
    if (!issuer) {
      float pm[8];
      fold_import(pm);
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        float p = fmaf(cc, pm[j], cb * Areg[j]);
        if (8 * fch + j == frow) p += ca;
        pm[j] = p;
      }
      uint4 hi, lo;
      split8(pm, hi, lo);
      *reinterpret_cast<uint4*>(PH + sw128_off(frow, fch)) = hi;
      *reinterpret_cast<uint4*>(PL + sw128_off(frow, fch)) = lo;
    }
    end_phase();
    // ---------------- X <- X Pm ----------------
    if (lead) {
      for (int mb = 0; mb < nblk; ++mb) {
        const uint32_t d = tb + C_X + 128 * mb;
        const uint64_t a_h = d_xh_k + mb * 1024, a_l = d_xl_k + mb * 1024;   // 16 KB per 128-row block
#pragma unroll
        for (int k = 0; k < HD / 16; ++k) {
          umma_ss(d, a_h + 2 * k, d_p + 2 * k, idesc_k128, k > 0);   // [XH PH^T | XH PL^T]
          umma_ss(d, a_l + 2 * k, d_p + 2 * k, idesc_k64, 1);        // left half += XL PH^T
        }
      }
      tc_commit(&mma_bar);
    }
    if (!issuer) {
      wait_mma();
      float* stage = reinterpret_cast<float*>(smem);          // last iteration: fp32 [H][W_LD]
      for (int mb = 0; mb < nblk; ++mb) {
        uint32_t r0[16], r1[16];
        tmem_ld_x16(tb + lane_base + C_X + 128 * mb + 16 * cs, r0);
        tmem_ld_x16(tb + lane_base + C_X + 128 * mb + 64 + 16 * cs, r1);
        tc_wait_ld();
        const int row = mb * 128 + trow;
        float f[16];
#pragma unroll
        for (int j = 0; j < 16; ++j) f[j] = __uint_as_float(r0[j]) + __uint_as_float(r1[j]);
        if (!last) {
#pragma unroll
          for (int k = 0; k < 2; ++k) {
            const float v[8] = {f[8 * k], f[8 * k + 1], f[8 * k + 2], f[8 * k + 3],
                                f[8 * k + 4], f[8 * k + 5], f[8 * k + 6], f[8 * k + 7]};
            uint4 hi, lo;
            split8(v, hi, lo);
            *reinterpret_cast<uint4*>(XH + sw128_off(row, 2 * cs + k)) = hi;
            *reinterpret_cast<uint4*>(XL + sw128_off(row, 2 * cs + k)) = lo;
          }
        } else {
          // all MMAs that read the operand tiles have completed: reuse them as the fp32 staging
          float4* dst = reinterpret_cast<float4*>(stage + (size_t)row * W_LD + 16 * cs);
#pragma unroll
          for (int v = 0; v < 4; ++v) dst[v] = make_float4(f[4 * v], f[4 * v + 1], f[4 * v + 2], f[4 * v + 3]);
        }
      }
    }
    end_phase();
  }
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  // ---- coalesced write-out: fused commit W <- W - NS(g) (Eq. 8) or NS(g) -> G ----
  {
    const float* stage = reinterpret_cast<const float*>(smem);
    constexpr int WB = 4;
    for (int e0 = issuer ? n4 : tid; e0 < n4; e0 += THREADS * WB) {
      float4 w[WB];
#pragma unroll
      for (int u = 0; u < WB; ++u) {
        const int e = e0 + u * THREADS;
        w[u] = (Wm != nullptr && e < n4) ? reinterpret_cast<const float4*>(Wm + mat_off)[e]
                                         : make_float4(0.f, 0.f, 0.f, 0.f);
      }
#pragma unroll
      for (int u = 0; u < WB; ++u) {
        const int e = e0 + u * THREADS;
        if (e >= n4) continue;
        const int row = e >> 4, c = (e & 15) * 4;
        const float4 x = *reinterpret_cast<const float4*>(stage + (size_t)row * W_LD + c);
        if (Wm != nullptr) {
          w[u].x -= x.x; w[u].y -= x.y; w[u].z -= x.z; w[u].w -= x.w;
          reinterpret_cast<float4*>(Wm + mat_off)[e] = w[u];
          reinterpret_cast<uint2*>(Wb + mat_off)[e] =
              make_uint2(ttt_pack_wop2(w[u].x, w[u].y), ttt_pack_wop2(w[u].z, w[u].w));
        } else {
          reinterpret_cast<float4*>(X)[e] = x;
        }
      }
    }
  }
  if (warp == 0) tmem_dealloc(tb, tmem_cols);
}

int ns_tc_supported(const ttt_config* cfg) {
  if (ns_tc_wide_supported(cfg)) return 1;
  return cfg->act_dtype == TTT_BF16 && cfg->hd == 64 && cfg->hidden % 128 == 0 &&
         cfg->hidden >= 128 && cfg->hidden <= 512 && !cfg->linear_fast_weight;
}

// NS of all 3*nh matrices of the pending gradient (the partial sets are folded in first).
// fuse_commit: also apply W <- W - NS(g) (fp32 master + bf16 copy) and clear the pending set;
// otherwise NS(g) is left in G (G_valid) for the commit kernel.
int launch_ns_tc(ttt_ctx* ctx, bool fuse_commit, cudaStream_t s) {
  const ttt_config& c = ctx->cfg;
  if (c.hd == 128) return launch_ns_tc_wide(ctx, fuse_commit, s);
  size_t smem = (size_t)2 * c.hidden * 128 + 4 * 8192 + 128 * nstc::S_LD * sizeof(float);
  const size_t stage = (size_t)c.hidden * nstc::W_LD * sizeof(float);
  if (stage > smem) smem = stage;
  smem += 1024;
  if (smem > ctx->attr_smem_ns) {
    TTT_CUDA_TRY(ctx, cudaFuncSetAttribute(ns_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                           (int)smem), "ns_tc_kernel smem attr");
    ctx->attr_smem_ns = smem;
  }
  const uint32_t alloc = c.hidden <= 256 ? 256 : 512;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(3 * c.nh);
  cfg.blockDim = dim3(nstc::LAUNCH_THREADS);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = s;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  float* G = ctx->G;
  const float* P = ctx->partials;
  int n_sets = ctx->n_partials, use_G = ctx->G_valid ? 1 : 0, H = c.hidden, iters = c.ns_iters;
  size_t set_elems = 3 * ctx->mat_elems;
  float* Wm = fuse_commit ? ctx->Wm : nullptr;
  ttt_wop_t* Wb = fuse_commit ? ctx->Wb : nullptr;
  cudaError_t e = cudaLaunchKernelEx(&cfg, ns_tc_kernel, G, P, n_sets, set_elems, use_G, H, iters, alloc, Wm, Wb);
  if (e != cudaSuccess) return set_error(ctx, TTT_ERR_CUDA, "ns_tc_kernel launch", e);
  TTT_LAUNCH_CHECK(ctx, "ns_tc_kernel");
  ctx->G_valid = !fuse_commit;
  ctx->n_partials = 0;
  return TTT_OK;
}

}  // namespace ttt
