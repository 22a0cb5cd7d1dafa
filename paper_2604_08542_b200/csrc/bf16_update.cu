// bf16_update.cu — fused tensor-core gradient kernel of the TTT update (steps 1-5 of the hot path,
// DESIGN.md "Kernels"; Eq. 8 with Eq. 9 and Eq. 12).
//
// Formulation ("hidden on lanes"): one CTA owns 128 hidden units of one head and a range of tokens.
// Everything is computed TRANSPOSED so that each MMA has M = 128 hidden units on the TMEM lanes:
//   forward   A^T  = W1^T K^T,  B^T = W3^T K^T,  g^T = W2 V^T      [128 x T]  (contract over hd)
//   epilogue  s = sigmoid(A); S = A s; Hd = S B; dHd = -eta g
//             dA = dHd B (s + S (1 - s)); dB = dHd S; Hd' = -eta Hd            (fp32 -> bf16)
//   gradient  G1^T += dA^T K,  G3^T += dB^T K,  G2 += Hd'^T V      [128 x hd] (contract over tokens)
// The A operand of every MMA lives in TMEM (weights: loaded once; dA/dB/Hd': written by the
// epilogue over their own fp32 sources), the B operand is the K or V token tile that TMA put in
// shared memory with the 128-byte swizzle; the SAME tile serves the forward MMA as a K-major
// operand and the gradient MMA as an MN-major operand. Gradient accumulators stay in TMEM for the
// CTA's whole token range; one fp32 partial per CTA goes to HBM/L2 and is summed in a fixed order
// by the commit kernel (deterministic, no float atomics).
//
// Warp roles (384 threads): warp 0 = TMA producer, warp 1 = MMA issuer, warp 2 = learning-rate
// loader (-eta of each tile into the stage's shared-memory slot), warps 4-7 / 8-11 = two epilogue
// warpgroups that alternate token tiles (TMEM accumulators are double-buffered). The epilogue math
// is packed fp32x2 (FFMA2/FMUL2): two tokens of one hidden unit per instruction.
#include <stdio.h>

#include "tc_common.cuh"
#include "ttt_internal.h"

#ifdef TTT_TRACE   // debug builds only: per-tile clock timeline of CTA (0,0,0), staged in smem
__device__ long long g_ttt_trace[64 * 16];
#define TTT_TR(i, k)                                                                  \
  do {                                                                                \
    if ((i) < 64 && blockIdx.x == 0 && blockIdx.y == 0 && blockIdx.z == 0)            \
      tr_s[(i) * 16 + (k)] = (unsigned)clock();                                       \
  } while (0)
extern "C" int ttt_debug_trace(long long* host) {
  return (int)cudaMemcpyFromSymbol(host, g_ttt_trace, sizeof(g_ttt_trace));
}
#else
#define TTT_TR(i, k) do { } while (0)
#endif

namespace ttt {

namespace upd {
constexpr int HS = 128;        // hidden units per CTA (MMA M)
constexpr int T = 32;          // tokens per tile (forward MMA N, gradient MMA K)
constexpr int STAGES = 6;      // K/V shared-memory ring
constexpr int THREADS = 384;
constexpr int TILE_BYTES = T * 128;  // one [T x 64] bf16 tile

// TMEM column plan for hd = 64 (512 columns x 128 lanes x 32 bit)
constexpr uint32_t C_W1 = 0, C_W3 = 32, C_W2 = 64;        // bf16 weights as A operands, 32 cols each
constexpr uint32_t C_G1 = 96, C_G3 = 160, C_G2 = 224;     // fp32 gradient accumulators, 64 cols each
constexpr uint32_t C_BUF = 288, BUF_STRIDE = 96;          // two forward buffers: A | B | g, 32 cols each
}  // namespace upd

template <bool LOSS>
__global__ void __launch_bounds__(upd::THREADS, 1)
bf16_update_kernel(const __grid_constant__ CUtensorMap mapK, const __grid_constant__ CUtensorMap mapV,
                   const __nv_bfloat16* __restrict__ Wb, const float* __restrict__ lr,
                   float* __restrict__ P, float* __restrict__ loss_part, int M, int nh, int H,
                   int tiles_total, int tiles_per_split) {
  using namespace upd;
  constexpr int HD = 64;
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) &
                                             ~static_cast<uintptr_t>(1023));
  __shared__ uint64_t full[STAGES], empty[STAGES], fwd_full[2], epi_done[2], w_ready, grad_done;
  __shared__ uint32_t tmem_base_s;
  __shared__ float loss_red[8];
  __shared__ __align__(16) float ne_s[STAGES][T];   // -eta of the stage's tokens (0 beyond M)
#ifdef TTT_TRACE
  __shared__ unsigned tr_s[64 * 16];
  for (int e = threadIdx.x; e < 64 * 16; e += blockDim.x) tr_s[e] = 0;
  __syncthreads();
  if (threadIdx.x == 0) tr_s[15] = (unsigned)clock();
#endif

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int split = blockIdx.x, slice = blockIdx.y, h = blockIdx.z;
  const int nslices = gridDim.y;
  const int tile_lo = split * tiles_per_split;
  const int ntiles = min(tiles_per_split, tiles_total - tile_lo);

  if (tid == 0) {
    for (int s = 0; s < STAGES; ++s) { mbar_init(&full[s], 2); mbar_init(&empty[s], 1); }
    for (int b = 0; b < 2; ++b) { mbar_init(&fwd_full[b], 1); mbar_init(&epi_done[b], 8); }
    mbar_init(&w_ready, 4);
    mbar_init(&grad_done, 1);
    fence_mbar_init();
  }
  if (warp == 0) { tmem_alloc(&tmem_base_s, 512); tmem_relinquish(); }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tb = tmem_base_s;
  if (tid == 0) TTT_TR(0, 14);

  if (warp == 0) {
    // ===================== TMA producer =====================
    if (elect_one()) {
      tma_prefetch_desc(&mapK);
      tma_prefetch_desc(&mapV);
      for (int i = 0; i < ntiles; ++i) {
        const int s = i % STAGES, it = i / STAGES;
        mbar_wait(&empty[s], (it & 1) ^ 1);
        TTT_TR(i, 12);
        mbar_arrive_expect_tx(&full[s], 2 * TILE_BYTES);
        uint8_t* dst = smem + s * 2 * TILE_BYTES;
        tma_load_2d(dst, &mapK, &full[s], h * HD, (tile_lo + i) * T);
        tma_load_2d(dst + TILE_BYTES, &mapV, &full[s], h * HD, (tile_lo + i) * T);
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer =====================
    if (elect_one()) {
      constexpr uint32_t idesc_f = umma_idesc_bf16(HS, T, 0, 0);    // B = token tile, K-major
      constexpr uint32_t idesc_g = umma_idesc_bf16(HS, HD, 0, 1);   // B = token tile, MN-major
      const uint32_t smem_base = smem_u32(smem);
      mbar_wait(&w_ready, 0);
      tc_fence_after();
      auto fwd = [&](int i) {
        const int s = i % STAGES, it = i / STAGES, b = i & 1;
        TTT_TR(i, 0);
        mbar_wait(&full[s], it & 1);
        tc_fence_after();
        TTT_TR(i, 1);
        const uint32_t ks = smem_base + s * 2 * TILE_BYTES, vs = ks + TILE_BYTES;
        const uint32_t acc = tb + C_BUF + b * BUF_STRIDE;
#pragma unroll
        for (int k = 0; k < HD / 16; ++k)
          umma_ts(acc, tb + C_W1 + 8 * k, umma_smem_desc_sw128(ks + 32 * k, 16, 1024), idesc_f, k > 0);
#pragma unroll
        for (int k = 0; k < HD / 16; ++k)
          umma_ts(acc + 32, tb + C_W3 + 8 * k, umma_smem_desc_sw128(ks + 32 * k, 16, 1024), idesc_f, k > 0);
#pragma unroll
        for (int k = 0; k < HD / 16; ++k)
          umma_ts(acc + 64, tb + C_W2 + 8 * k, umma_smem_desc_sw128(vs + 32 * k, 16, 1024), idesc_f, k > 0);
        tc_commit(&fwd_full[b]);
        TTT_TR(i, 2);
      };
      auto grad = [&](int i) {
        const int s = i % STAGES, b = i & 1, n = i >> 1;
        mbar_wait(&epi_done[b], n & 1);
        tc_fence_after();
        TTT_TR(i, 3);
        const uint32_t ks = smem_base + s * 2 * TILE_BYTES, vs = ks + TILE_BYTES;
        const uint32_t opnd = tb + C_BUF + b * BUF_STRIDE;   // dA | dB | Hd' alias A | B | g
#pragma unroll
        for (int k = 0; k < T / 16; ++k)
          umma_ts(tb + C_G1, opnd + 24 * k, umma_smem_desc_sw128(ks + 2048 * k, TILE_BYTES, 1024),
                  idesc_g, (i > 0 || k > 0));
#pragma unroll
        for (int k = 0; k < T / 16; ++k)
          umma_ts(tb + C_G3, opnd + 32 + 24 * k, umma_smem_desc_sw128(ks + 2048 * k, TILE_BYTES, 1024),
                  idesc_g, (i > 0 || k > 0));
#pragma unroll
        for (int k = 0; k < T / 16; ++k)
          umma_ts(tb + C_G2, opnd + 64 + 24 * k, umma_smem_desc_sw128(vs + 2048 * k, TILE_BYTES, 1024),
                  idesc_g, (i > 0 || k > 0));
        tc_commit(&empty[s]);
        TTT_TR(i, 4);
      };
      if (ntiles > 0) fwd(0);
      for (int i = 0; i < ntiles; ++i) {
        if (i + 1 < ntiles) fwd(i + 1);
        grad(i);
      }
      tc_commit(&grad_done);
    }
  } else if (warp == 2) {
    // ===================== learning-rate loader =====================
    // -eta of tile i (32 tokens = one 128-B line of lr) goes to the stage's shared-memory slot.
    // The global loads run LRPF tiles ahead of the ring (register double buffer), so their
    // latency is never on the critical path of a tile.
    constexpr int LRPF = 8;
    const float* lrh = lr + (size_t)h * M;
    auto ld_batch = [&](int i0, float (&v)[LRPF]) {
#pragma unroll
      for (int u = 0; u < LRPF; ++u) {
        const int t = (tile_lo + i0 + u) * T + lane;
        v[u] = (i0 + u < ntiles && t < M) ? -__ldg(lrh + t) : 0.f;
      }
    };
    float cur[LRPF], nxt[LRPF];
    ld_batch(0, cur);
    for (int i0 = 0; i0 < ntiles; i0 += LRPF) {
      ld_batch(i0 + LRPF, nxt);
#pragma unroll
      for (int u = 0; u < LRPF; ++u) {
        const int i = i0 + u;
        if (i < ntiles) {
          const int s = i % STAGES, it = i / STAGES;
          mbar_wait(&empty[s], (it & 1) ^ 1);
          ne_s[s][lane] = cur[u];
          __syncwarp();
          if (lane == 0) mbar_arrive(&full[s]);
        }
      }
#pragma unroll
      for (int u = 0; u < LRPF; ++u) cur[u] = nxt[u];
    }
  } else if (warp >= 4) {
    // ===================== epilogue warpgroups =====================
    const int wg = (warp - 4) >> 2, q = warp & 3;
    const int j = q * 32 + lane;                       // hidden unit within the slice = TMEM lane
    const uint32_t lane_base = static_cast<uint32_t>(q * 32) << 16;
    const size_t me = (size_t)nh * H * HD;
    const size_t row = ((size_t)h * H + (size_t)slice * HS + j) * HD;
    if (wg == 0) {
      // weights -> TMEM as A operands: row j of W1^T, W3^T, W2 (64 bf16 = 32 words each);
      // all 24 loads are issued before the first TMEM store
      const uint32_t cols[3] = {C_W1, C_W2, C_W3};
      uint4 x[3][8];
#pragma unroll
      for (int mat = 0; mat < 3; ++mat) {
        const uint4* src = reinterpret_cast<const uint4*>(Wb + mat * me + row);
#pragma unroll
        for (int v = 0; v < 8; ++v) x[mat][v] = __ldg(src + v);
      }
#pragma unroll
      for (int mat = 0; mat < 3; ++mat) {
        uint32_t r[32];
#pragma unroll
        for (int v = 0; v < 8; ++v) {
          r[4 * v] = x[mat][v].x; r[4 * v + 1] = x[mat][v].y;
          r[4 * v + 2] = x[mat][v].z; r[4 * v + 3] = x[mat][v].w;
        }
        tmem_st_x32(tb + lane_base + cols[mat], r);
      }
      tc_wait_st();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&w_ready);
    }
    uint64_t loss2 = 0ull;
    const uint64_t HALF2 = pack2(0.5f, 0.5f), NHALF2 = pack2(-0.5f, -0.5f);
    for (int i = 0; i < ntiles; ++i) {
      // both warpgroups work on every tile: warpgroup `wg` owns token columns [16 wg, 16 wg + 16)
      const int b = i & 1, n = i >> 1, s = i % STAGES;
      const uint32_t buf = tb + lane_base + C_BUF + b * BUF_STRIDE;
      if (q == 0 && lane == 0) TTT_TR(i, 5 + wg);
      mbar_wait(&fwd_full[b], n & 1);
      mbar_wait(&full[s], (i / STAGES) & 1);     // direct acquire of the loader's -eta slot
      tc_fence_after();
      if (q == 0 && lane == 0) TTT_TR(i, 7 + wg);
      const uint2* nes = reinterpret_cast<const uint2*>(&ne_s[s][0]);
      uint32_t ra[16], rb[16], rg[16];
      tmem_ld_x16(buf + 16 * wg, ra);
      tmem_ld_x16(buf + 32 + 16 * wg, rb);
      tmem_ld_x16(buf + 64 + 16 * wg, rg);
      tc_wait_ld();
      uint32_t pa[8], pb[8], ph[8];
#pragma unroll
      for (int c = 0; c < 16; c += 2) {
        const uint64_t a = pack2u(ra[c], ra[c + 1]);
        const uint64_t bb = pack2u(rb[c], rb[c + 1]);
        const uint64_t g = pack2u(rg[c], rg[c + 1]);
        const uint2 nev = nes[8 * wg + (c >> 1)];
        const uint64_t ne = pack2u(nev.x, nev.y);
        // sigmoid(a) = 0.5 tanh(a/2) + 0.5 on the MUFU; 1 - sigmoid = 0.5 - 0.5 tanh(a/2)
        float x0, x1;
        unpack2(fmul2(a, HALF2), x0, x1);
        const uint64_t th = pack2(tanh_approx(x0), tanh_approx(x1));
        const uint64_t sg = ffma2(th, HALF2, HALF2);
        const uint64_t om = ffma2(th, NHALF2, HALF2);
        const uint64_t S = fmul2(a, sg);                 // SiLU(a)
        const uint64_t t2 = ffma2(S, om, sg);            // SiLU'(a) = s + S (1 - s)
        const uint64_t hdv = fmul2(S, bb);               // hidden activation Hd
        const uint64_t dhd = fmul2(ne, g);               // dHd = (-eta v) W2^T
        pa[c >> 1] = pack_bf16x2_from2(fmul2(fmul2(dhd, bb), t2));   // dA
        pb[c >> 1] = pack_bf16x2_from2(fmul2(dhd, S));               // dB
        ph[c >> 1] = pack_bf16x2_from2(fmul2(ne, hdv));              // Hd' = -eta Hd
        if (LOSS) loss2 = ffma2(hdv, dhd, loss2);
      }
      // bf16 operands overwrite fp32 columns this warp itself has just read: tokens [16 wg, +16)
      // of dA / dB / Hd' go to columns [24 wg, 24 wg + 8) of the A / B / g regions
      tmem_st_x8(buf + 24 * wg, pa);
      tmem_st_x8(buf + 32 + 24 * wg, pb);
      tmem_st_x8(buf + 64 + 24 * wg, ph);
      tc_wait_st();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&epi_done[b]);
      if (q == 0 && lane == 0) TTT_TR(i, 9 + wg);
    }
    // ---- flush the gradient accumulators: one fp32 partial slice per CTA ----
    if (warp == 4 && lane == 0) TTT_TR(2, 13);
    mbar_wait(&grad_done, 0);
    tc_fence_after();
    if (warp == 4 && lane == 0) TTT_TR(2, 14);
    float* Pset = P + (size_t)split * 3 * me;
    auto flush = [&](uint32_t col, int mat, int c0, int ncols) {
      float4* dst = reinterpret_cast<float4*>(Pset + mat * me + row + c0);
      for (int c = 0; c < ncols; c += 16) {
        uint32_t r[16];
        if (ntiles > 0) {
          tmem_ld_x16(tb + lane_base + col + c0 + c, r);
          tc_wait_ld();
        } else {
#pragma unroll
          for (int u = 0; u < 16; ++u) r[u] = 0u;
        }
#pragma unroll
        for (int v = 0; v < 4; ++v)
          dst[(c >> 2) + v] = make_float4(__uint_as_float(r[4 * v]), __uint_as_float(r[4 * v + 1]),
                                          __uint_as_float(r[4 * v + 2]), __uint_as_float(r[4 * v + 3]));
      }
    };
    if (wg == 0) { flush(C_G1, 0, 0, 64); flush(C_G2, 1, 0, 32); }
    else         { flush(C_G3, 2, 0, 64); flush(C_G2, 1, 32, 32); }
    if (warp == 4 && lane == 0) TTT_TR(2, 15);
    if (LOSS) {
      float l0, l1;
      unpack2(loss2, l0, l1);
      float loss = l0 + l1;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) loss += __shfl_xor_sync(0xffffffffu, loss, o);
      if (lane == 0) loss_red[warp - 4] = loss;
      asm volatile("bar.sync 1, 256;" ::: "memory");
      if (warp == 4 && lane == 0) {
        float t = 0.f;
        for (int w = 0; w < 8; ++w) t += loss_red[w];
        loss_part[((size_t)split * nslices + slice) * nh + h] = t;
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 0) tmem_dealloc(tb, 512);
#ifdef TTT_TRACE
  if (threadIdx.x == 0) tr_s[16 + 15] = (unsigned)clock();
  __syncthreads();
  if (blockIdx.x == 0 && blockIdx.y == 0 && blockIdx.z == 0)
    for (int e = threadIdx.x; e < 64 * 16; e += blockDim.x) g_ttt_trace[e] = tr_s[e];
#endif
}

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------
typedef CUresult (*encode_tiled_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*,
                                    const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                    const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                    CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// 2-D bf16 tensor [rows][cols] (row stride ld elements), box = [box_rows][64 cols], 128-B swizzle.
// Out-of-bounds rows are zero-filled, which makes the ragged last token tile contribute nothing.
int make_token_map(ttt_ctx* ctx, CUtensorMap* map, const void* base, int64_t rows, int64_t cols,
                   int64_t ld, int box_rows) {
  cuuint64_t gdim[2] = {(cuuint64_t)cols, (cuuint64_t)rows};
  cuuint64_t gstr[1] = {(cuuint64_t)ld * 2};
  cuuint32_t box[2] = {64, (cuuint32_t)box_rows};
  cuuint32_t estr[2] = {1, 1};
  CUresult r = reinterpret_cast<encode_tiled_fn>(ctx->encode_tiled)(
      map, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), gdim, gstr, box, estr,
      CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
      CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    snprintf(ctx->err, sizeof(ctx->err), "cuTensorMapEncodeTiled failed (CUresult %d)", (int)r);
    return TTT_ERR_CUDA;
  }
  return TTT_OK;
}

static void update_split(const ttt_ctx* ctx, int64_t M, int* tiles_total, int* tiles_per_split,
                         int* splits) {
  const int tiles = (int)((M + upd::T - 1) / upd::T);
  const int pairs = ctx->cfg.nh * (ctx->cfg.hidden / upd::HS);
  int want = ctx->sm_count / pairs;           // one wave of CTAs, one CTA per SM
  if (want < 1) want = 1;
  if (want > tiles) want = tiles;
  const int tps = (tiles + want - 1) / want;
  *tiles_total = tiles;
  *tiles_per_split = tps;
  *splits = (tiles + tps - 1) / tps;
}

int bf16_partials_needed(const ttt_ctx* ctx, int64_t M) {
  int a, b, s;
  update_split(ctx, M, &a, &b, &s);
  return s;
}

int bf16_supported(const ttt_config* cfg, char* why, size_t why_len) {
  if (cfg->hd != 64) { snprintf(why, why_len, "bf16 path: hd must be 64 (got %d)", cfg->hd); return 0; }
  if (cfg->hidden % 128 != 0 || cfg->hidden < 128 || cfg->hidden > 256) {
    snprintf(why, why_len, "bf16 path: hidden must be 128 or 256 (got %d)", cfg->hidden);
    return 0;
  }
  if (cfg->linear_fast_weight) { snprintf(why, why_len, "bf16 path: linear test mode is f32-only"); return 0; }
  return 1;
}

int bf16_accumulate(ttt_ctx* ctx, const __nv_bfloat16* K, const __nv_bfloat16* V, const float* lr,
                    int64_t M, int64_t ld, bool want_loss, int* used, int* loss_rows,
                    cudaStream_t s) {
  const ttt_config& c = ctx->cfg;
  int tiles, tps, splits;
  update_split(ctx, M, &tiles, &tps, &splits);
  CUtensorMap mapK, mapV;
  int rc = make_token_map(ctx, &mapK, K, M, (int64_t)c.nh * c.hd, ld, upd::T);
  if (rc != TTT_OK) return rc;
  rc = make_token_map(ctx, &mapV, V, M, (int64_t)c.nh * c.hd, ld, upd::T);
  if (rc != TTT_OK) return rc;
  const size_t smem = (size_t)upd::STAGES * 2 * upd::TILE_BYTES + 1024;
  static bool attr_set = false;
  if (!attr_set) {
    TTT_CUDA_TRY(ctx, cudaFuncSetAttribute(bf16_update_kernel<false>,
                                           cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem),
                 "bf16_update_kernel smem attr");
    TTT_CUDA_TRY(ctx, cudaFuncSetAttribute(bf16_update_kernel<true>,
                                           cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem),
                 "bf16_update_kernel smem attr");
    attr_set = true;
  }
  const int nslices = c.hidden / upd::HS;
  float* P = ctx->partials + (size_t)ctx->n_partials * 3 * ctx->mat_elems;
  dim3 grid(splits, nslices, c.nh);
  if (want_loss)
    bf16_update_kernel<true><<<grid, upd::THREADS, smem, s>>>(mapK, mapV, ctx->Wb, lr, P,
                                                             ctx->loss_part, (int)M, c.nh,
                                                             c.hidden, tiles, tps);
  else
    bf16_update_kernel<false><<<grid, upd::THREADS, smem, s>>>(mapK, mapV, ctx->Wb, lr, P,
                                                              ctx->loss_part, (int)M, c.nh,
                                                              c.hidden, tiles, tps);
  TTT_LAUNCH_CHECK(ctx, "bf16_update_kernel");
  *used = splits;
  *loss_rows = splits * nslices;
  return TTT_OK;
}

}  // namespace ttt
