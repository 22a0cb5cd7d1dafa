// bf16_apply_wide.cu — fast-weight apply O = (SiLU(Q W1) * (Q W3)) W2 for head dimension 128
// (Eq. 12 on the query tokens), tcgen05 / TMEM / TMA.
//
// Tokens on the 128 TMEM lanes as in bf16_apply.cu. At hd = 128 a head's weights (3 x H x 128 bf16,
// 393 KB at H = 512) no longer fit in shared memory, so they are streamed: a persistent CTA takes
// units of (head, two 128-token tiles), keeps both Q tiles in shared memory and both O
// accumulators in TMEM, and walks the hidden dimension in steps of 64 units through a ring of
// weight stages ([W1^T | W3^T] rows as one N = 128 B operand, W2 rows as the MN-major B operand of
// the down projection). Every streamed weight byte is used by 256 tokens.
//   TMEM (512 columns): O(t) fp32 [128 x 128] at 128 t; forward accumulators x | b of tile t
//   (64 + 64 columns) at 256 + 128 t; the bf16 hidden activation Hq (A operand of the down MMAs)
//   overwrites the first 32 columns of its own x once every epilogue warp of the tile holds its
//   x | b in registers. (Q as a TMEM operand with 32-hidden steps was built and measured: the
//   F -> epilogue -> D -> F chain of a tile is latency-bound and the shorter steps lose, 147 vs 131 us.)
//   MMA order per step n: D(0,n) F(0,n+1) D(1,n) F(1,n+1) — the forward MMAs of one tile run while
//   the other tile's epilogue works; in-order execution makes the re-use of x safe.
//   Warps: TMA producer, MMA issuer, two epilogue groups of 8 warps, one per tile (SwiGLU
//   epilogue per step, O -> bf16 -> global).
#include <stdio.h>
#include <stdlib.h>

#include "tc_common.cuh"
#include "ttt_internal.h"

namespace ttt {

int make_token_map(ttt_ctx* ctx, CUtensorMap* map, const void* base, int64_t rows, int64_t cols,
                   int64_t ld, int box_rows);   // bf16_update.cu

namespace appw {
constexpr int HD = 128;        // head dimension
constexpr int TM = 128;        // tokens per tile (MMA M)
constexpr int HSTEP = 64;      // hidden units per step
constexpr int NST = 3;         // weight ring stages
constexpr int GRP_WARPS = 8;   // epilogue warps per tile
constexpr int THREADS = (4 + 2 * GRP_WARPS) * 32;
constexpr int QSUB_BYTES = TM * 128;            // [128 tokens x 64] bf16 sub-tile (half of hd)
constexpr int QTILE_BYTES = 2 * QSUB_BYTES;
constexpr int BOX_BYTES = HSTEP * 128;          // one TMA box of weights: [64 rows x 64]
constexpr int FSUB_BYTES = 2 * BOX_BYTES;       // [W1^T rows | W3^T rows] x one hd half
constexpr int W2_OFF = 2 * FSUB_BYTES;          // W2 rows of the step: two hd halves, BOX_BYTES each
constexpr int WSTAGE_BYTES = W2_OFF + 2 * BOX_BYTES;
constexpr size_t SMEM_BYTES = 2 * (size_t)QTILE_BYTES + (size_t)NST * WSTAGE_BYTES + 1024;
constexpr uint32_t C_O = 0, C_F = 256;
}  // namespace appw

__global__ void __launch_bounds__(appw::THREADS, 1)
bf16_apply_wide_kernel(const __grid_constant__ CUtensorMap mapW, const __grid_constant__ CUtensorMap mapQ,
                       __nv_bfloat16* __restrict__ O, int M, int64_t ld, int nh, int H, int npairs) {
  using namespace appw;
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  const uint32_t sbase = (smem_u32(smem_raw) + 1023u) & ~1023u;
  uint8_t* smem = smem_raw + (sbase - smem_u32(smem_raw));
  uint8_t* wring = smem + 2 * QTILE_BYTES;
  __shared__ uint64_t w_full[NST], w_empty[NST], q_full[2], q_free[2], f_full[2], hq_ready[2],
      o_full[2], o_free[2];
  __shared__ uint32_t tmem_base_s;

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int nstep = H / HSTEP;
  const int nunits = nh * npairs;

  if (tid == 0) {
    for (int s = 0; s < NST; ++s) { mbar_init(&w_full[s], 1); mbar_init(&w_empty[s], 1); }
    for (int t = 0; t < 2; ++t) {
      mbar_init(&q_full[t], 1);
      mbar_init(&q_free[t], 1);
      mbar_init(&f_full[t], 1);
      mbar_init(&hq_ready[t], GRP_WARPS);
      mbar_init(&o_full[t], 1);
      mbar_init(&o_free[t], GRP_WARPS);
    }
    fence_mbar_init();
    tma_prefetch_desc(&mapW);
    tma_prefetch_desc(&mapQ);
  }
  if (warp == 0) { tmem_alloc(&tmem_base_s, 512); tmem_relinquish(); }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tb = tmem_base_s;
  if (tb != 0) __trap();      // all 512 columns belong to this CTA: absolute columns below
  // programmatic dependent launch: everything above overlapped the tail of the commit kernel
  asm volatile("griddepcontrol.wait;" ::: "memory");

  if (warp == 0) {
    // ===================== TMA producer =====================
    if (elect_one()) {
      int g = 0;
      for (int u = 0, unit = blockIdx.x; unit < nunits; unit += gridDim.x, ++u) {
        const int h = unit / npairs, p = unit % npairs;
        for (int t = 0; t < 2; ++t) {
          if (u > 0) mbar_wait(&q_free[t], (u - 1) & 1);     // the forward MMAs of the tile's previous unit are done
          mbar_arrive_expect_tx(&q_full[t], QTILE_BYTES);
          for (int c = 0; c < 2; ++c)
            tma_load_2d(smem + t * QTILE_BYTES + c * QSUB_BYTES, &mapQ, &q_full[t], h * HD + c * 64,
                        (2 * p + t) * TM);
        }
        for (int n = 0; n < nstep; ++n, ++g) {
          const int s = g % NST;
          if (g >= NST) mbar_wait(&w_empty[s], ((g / NST) & 1) ^ 1);
          mbar_arrive_expect_tx(&w_full[s], WSTAGE_BYTES);
          uint8_t* dst = wring + s * WSTAGE_BYTES;
          const int r1 = (0 * nh + h) * H + n * HSTEP, r2 = (1 * nh + h) * H + n * HSTEP,
                    r3 = (2 * nh + h) * H + n * HSTEP;
          for (int c = 0; c < 2; ++c) {
            tma_load_2d(dst + c * FSUB_BYTES, &mapW, &w_full[s], c * 64, r1);
            tma_load_2d(dst + c * FSUB_BYTES + BOX_BYTES, &mapW, &w_full[s], c * 64, r3);
            tma_load_2d(dst + W2_OFF + c * BOX_BYTES, &mapW, &w_full[s], c * 64, r2);
          }
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer =====================
    if (elect_one()) {
      constexpr uint32_t idesc_f = umma_idesc(TM, 2 * HSTEP, 0, 0, TTT_FMT_BF16, TTT_FMT_BF16);   // A = Q (smem), B = [W1^T | W3^T] rows
      const uint64_t dq = umma_smem_desc_sw128(sbase, 16, 1024);
      constexpr uint32_t idesc_d = umma_idesc(TM, HD, 0, 1, TTT_FMT_BF16, TTT_FMT_BF16);          // A = Hq (TMEM), B = W2 rows, MN-major
      const uint64_t dwf = umma_smem_desc_sw128(sbase + 2 * QTILE_BYTES, 16, 1024);
      const uint64_t dw2 = umma_smem_desc_sw128(sbase + 2 * QTILE_BYTES + W2_OFF, BOX_BYTES, 1024);
      auto issueF = [&](int t, int s) {      // x | b of tile t <- Q(t) [W1^T | W3^T]^T of ring stage s
#pragma unroll
        for (int k = 0; k < HD / 16; ++k) {
          const uint64_t a = dq + (uint64_t)(t * (QTILE_BYTES >> 4) + (k >> 2) * (QSUB_BYTES >> 4) + (k & 3) * 2);
          const uint64_t b = dwf + (uint64_t)(s * (WSTAGE_BYTES >> 4) + (k >> 2) * (FSUB_BYTES >> 4) + (k & 3) * 2);
          umma_ss(C_F + t * 128, a, b, idesc_f, k > 0);
        }
        tc_commit(&f_full[t]);
      };
      auto issueD = [&](int t, int s, uint32_t acc) {   // O(t) (+)= Hq(t) W2[step rows]
#pragma unroll
        for (int k = 0; k < HSTEP / 16; ++k)             // +2048 B per 16 hidden rows
          umma_ts(C_O + t * 128, C_F + t * 128 + 8 * k,
                  dw2 + (uint64_t)(s * (WSTAGE_BYTES >> 4) + 128 * k), idesc_d, acc | k);
      };
      int g = 0;
      for (int u = 0, unit = blockIdx.x; unit < nunits; unit += gridDim.x, ++u) {
        mbar_wait(&w_full[g % NST], (g / NST) & 1);
        for (int t = 0; t < 2; ++t) {
          mbar_wait(&q_full[t], u & 1);
          tc_fence_after();
          issueF(t, g % NST);
          if (nstep == 1) tc_commit(&q_free[t]);
        }
        for (int n = 0; n < nstep; ++n, ++g) {
          const int s = g % NST, s1 = (g + 1) % NST;
          for (int t = 0; t < 2; ++t) {
            if (n == 0 && u > 0) mbar_wait(&o_free[t], (u - 1) & 1);   // previous O(t) has been read
            mbar_wait(&hq_ready[t], (u * nstep + n) & 1);
            tc_fence_after();
            issueD(t, s, n > 0);
            if (n == nstep - 1) tc_commit(&o_full[t]);
            if (t == 1) tc_commit(&w_empty[s]);
            if (n + 1 < nstep) {
              if (t == 0) { mbar_wait(&w_full[s1], ((g + 1) / NST) & 1); tc_fence_after(); }
              issueF(t, s1);
              if (n + 2 == nstep) tc_commit(&q_free[t]);
            }
          }
        }
      }
    }
  } else if (warp >= 4) {
    // ===================== epilogue warps: group t = one token tile =====================
    const int ew = warp - 4, t = ew >> 3, q = warp & 3, cg = (ew >> 2) & 1;   // tile, lane quadrant, column half
    const uint32_t lane_base = static_cast<uint32_t>(q * 32) << 16;
    const int row = q * 32 + lane;                         // token row of the tile = TMEM lane
    const uint64_t HALF2 = pack2(0.5f, 0.5f);
    const uint32_t buf = lane_base + C_F + t * 128;
    for (int u = 0, unit = blockIdx.x; unit < nunits; unit += gridDim.x, ++u) {
      const int h = unit / npairs, p = unit % npairs;
      for (int n = 0; n < nstep; ++n) {
        mbar_wait(&f_full[t], (u * nstep + n) & 1);
        tc_fence_after();
        uint32_t rx[32], rb[32];
        tmem_ld_x32(buf + 32 * cg, rx);
        tmem_ld_x32(buf + 64 + 32 * cg, rb);
        tc_wait_ld();
        tc_fence_before();
        // every warp of the tile holds its x | b: x may be overwritten (named barrier 1 + t, 8 warps)
        asm volatile("bar.sync %0, 256;" ::"r"(1 + t) : "memory");
        uint32_t ph[16];
#pragma unroll
        for (int c = 0; c < 32; c += 2) {
          const uint64_t x = fmul2(pack2u(rx[c], rx[c + 1]), HALF2);   // a / 2
          float x0, x1;
          unpack2(x, x0, x1);
          const uint64_t th = pack2(tanh_approx(x0), tanh_approx(x1));
          const uint64_t S = ffma2(x, th, x);                          // SiLU(a) = a/2 (1 + tanh(a/2))
          ph[c >> 1] = pack_bf16x2_from2(fmul2(S, pack2u(rb[c], rb[c + 1])));
        }
        tmem_st_x16(buf + 16 * cg, ph);
        tc_wait_st();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(&hq_ready[t]);
      }
      // ---- O(t) -> bf16 -> global: this thread owns token row `row`, columns 64 cg .. 64 cg + 63 ----
      mbar_wait(&o_full[t], u & 1);
      tc_fence_after();
      const int64_t tok = (int64_t)(2 * p + t) * TM + row;
#pragma unroll
      for (int half = 0; half < 2; ++half) {
        uint32_t ro[32];
        tmem_ld_x32(lane_base + C_O + t * 128 + 64 * cg + 32 * half, ro);
        tc_wait_ld();
        if (half == 1) {
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(&o_free[t]);
        }
        if (tok < M) {
          uint4* dst = reinterpret_cast<uint4*>(O + tok * ld + h * HD + 64 * cg + 32 * half);
#pragma unroll
          for (int v = 0; v < 4; ++v) {
            uint4 w;
            w.x = pack_bf16x2(__uint_as_float(ro[8 * v]), __uint_as_float(ro[8 * v + 1]));
            w.y = pack_bf16x2(__uint_as_float(ro[8 * v + 2]), __uint_as_float(ro[8 * v + 3]));
            w.z = pack_bf16x2(__uint_as_float(ro[8 * v + 4]), __uint_as_float(ro[8 * v + 5]));
            w.w = pack_bf16x2(__uint_as_float(ro[8 * v + 6]), __uint_as_float(ro[8 * v + 7]));
            dst[v] = w;
          }
        }
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 0) tmem_dealloc(tb, 512);
}

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------
int bf16_apply_wide_supported(const ttt_config* cfg) {
  return cfg->hd == appw::HD && cfg->hidden % appw::HSTEP == 0 && !cfg->linear_fast_weight;
}

int bf16_apply_wide(ttt_ctx* ctx, const __nv_bfloat16* Q, __nv_bfloat16* O, int64_t M, int64_t ld,
                    cudaStream_t s) {
  const ttt_config& c = ctx->cfg;
  // CTA-pair kernel by default (bf16_apply_wide_pair.cu); TTT_APPLY_WIDE_PAIR=0 selects this file's
  // single-CTA kernel (kept for A/B measurements)
  static const int use_pair = [] { const char* e = getenv("TTT_APPLY_WIDE_PAIR"); return e ? atoi(e) : 1; }();
  if (use_pair) {
    const int rc = bf16_apply_wide_pair(ctx, Q, O, M, ld, s);
    if (rc != 1) return rc;          // 1 = the device cannot host a CTA pair: single-CTA kernel below
  }
  const int tiles = (int)((M + appw::TM - 1) / appw::TM);
  const int npairs = (tiles + 1) / 2;
  CUtensorMap mapW, mapQ;
  int rc = make_token_map(ctx, &mapW, ctx->Wq, (int64_t)3 * c.nh * c.hidden, c.hd, c.hd, appw::HSTEP);
  if (rc != TTT_OK) return rc;
  rc = make_token_map(ctx, &mapQ, Q, M, (int64_t)c.nh * c.hd, ld, appw::TM);
  if (rc != TTT_OK) return rc;
  static bool attr_set = false;
  if (!attr_set) {
    TTT_CUDA_TRY(ctx, cudaFuncSetAttribute(bf16_apply_wide_kernel,
                                           cudaFuncAttributeMaxDynamicSharedMemorySize,
                                           (int)appw::SMEM_BYTES), "bf16_apply_wide_kernel smem attr");
    attr_set = true;
  }
  int grid = c.nh * npairs;
  if (grid > ctx->sm_count) grid = ctx->sm_count;      // persistent CTAs, units round-robin
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(grid);
  cfg.blockDim = dim3(appw::THREADS);
  cfg.dynamicSmemBytes = appw::SMEM_BYTES;
  cfg.stream = s;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  int Mi = (int)M, nh = c.nh, H = c.hidden;
  cudaError_t e = cudaLaunchKernelEx(&cfg, bf16_apply_wide_kernel, mapW, mapQ, O, Mi, ld, nh, H, npairs);
  if (e != cudaSuccess) return set_error(ctx, TTT_ERR_CUDA, "bf16_apply_wide_kernel launch", e);
  TTT_LAUNCH_CHECK(ctx, "bf16_apply_wide_kernel");
  return TTT_OK;
}

}  // namespace ttt
