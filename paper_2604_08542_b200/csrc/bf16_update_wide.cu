// bf16_update_wide.cu — fused fast-weight gradient kernel for head dimension 128 (tcgen05 / TMEM / TMA).
//
// Same computation as bf16_update.cu (Eq. 11-13: forward through the SwiGLU fast weights on
// the chunk's keys, gradient of the dot-product loss w.r.t. W1, W2, W3 with the per-token learning
// rate folded in), same orientation (hidden units on the 128 TMEM lanes, tokens on the MMA N / K
// axis), for hd = 128, where the TMEM budget is different: the three fp32 gradient accumulators of a
// 128-hidden slice take 3 x 128 = 384 of the 512 columns, so
//   * the weights stay in shared memory (A operands of SS-mode MMAs, 96 KB per slice),
//   * the forward accumulators x | b | g of one 32-token tile are single-buffered (96 columns),
//   * the fp16 operand Hd' of the W2 gradient re-uses the columns of x; the MMA order
//     b(i+1) g(i+1) | G2(i) | x(i+1) | commit | G1(i) G3(i) keeps the tensor pipe busy while the epilogue
//     of tile i+1 loads its accumulators and makes the overwrite of x safe (MMAs of one thread execute
//     in issue order). Measured: the issuing thread is stalled by pipe back-pressure 80 % of the time,
//     i.e. the kernel is bound by the SS-mode forward products (M128 N32 K16 at ~56 clk each).
// A CTA works on one (head, 128-hidden slice) pair at a time; its partial gradients go to one partial
// set per segment, summed in set order by the commit (deterministic, no float atomics).
#include <stdio.h>

#include "tc_common.cuh"
#include "ttt_internal.h"

namespace ttt {

int make_token_map(ttt_ctx* ctx, CUtensorMap* map, const void* base, int64_t rows, int64_t cols,
                   int64_t ld, int box_rows);   // bf16_update.cu

namespace updw {
constexpr int HS = 128;        // hidden units per CTA (MMA M)
constexpr int HD = 128;        // head dimension (forward MMA K, gradient MMA N)
constexpr int T = 32;          // tokens per tile (forward MMA N, gradient MMA K)
constexpr int STAGES = 5;      // K/V shared-memory ring
constexpr int EPI_WARPS = 8;
constexpr int CVT_WARPS = 4;   // stage finishers: warps 2, 3 and the two warps after the epilogue warps
constexpr int THREADS = (4 + EPI_WARPS + CVT_WARPS - 2) * 32;
constexpr int SUB_BYTES = T * 128;          // one [T x 64] bf16 sub-tile (half of hd), 128-B swizzled
constexpr int TILE_BYTES = 2 * SUB_BYTES;   // K or V tile
constexpr int STAGE_BYTES = 2 * TILE_BYTES;
constexpr int WSUB_BYTES = HS * 128;        // one [128 x 64] fp16 weight sub-tile
constexpr int WMAT_BYTES = 2 * WSUB_BYTES;
constexpr int W_BYTES = 3 * WMAT_BYTES;
constexpr int SLD = 64 + 4;                 // flush staging row stride (floats)
constexpr int STG_BYTES = HS * SLD * 4;     // [128][68] fp32 staging of one 64-column half
constexpr size_t SMEM_BYTES = (size_t)W_BYTES + (size_t)STAGES * STAGE_BYTES + STG_BYTES + 1024;

// TMEM column plan (512 columns x 128 lanes x 32 bit)
constexpr uint32_t C_G1 = 0, C_G3 = 128, C_G2 = 256;   // fp32 gradient accumulators [hidden][hd]
constexpr uint32_t C_X = 384, C_B = 416, C_G = 448;    // fp32 forward accumulators [hidden][token]
constexpr uint32_t C_OA = 480, C_OB = 496;             // fp16 operands 2 dA, dB [hidden][token], 16 cols
constexpr uint32_t C_OH = C_X;                         // fp16 operand Hd' = -eta Hd, over the dead x
}  // namespace updw

// Work distribution: the (head, slice) pairs x 32-token tiles form one list of units, pair-major; CTA c
// of `gridDim.x` takes units [c U / n, (c + 1) U / n) — every SM gets the same amount of work, and a
// CTA whose range crosses a pair boundary runs one segment per pair (weights reloaded, accumulators
// flushed in between). Segment j of a pair (in CTA order) writes partial set j; the pair's last
// segment zero-fills the sets up to `nsets`, so the commit sums the same number of sets everywhere.
template <bool LOSS>
__global__ void __launch_bounds__(updw::THREADS, 1)
bf16_update_wide_kernel(const __grid_constant__ CUtensorMap mapK, const __grid_constant__ CUtensorMap mapV,
                        const __grid_constant__ CUtensorMap mapW, const float* __restrict__ lr,
                        float* __restrict__ P, float* __restrict__ loss_part, int M, int nh, int H,
                        int tiles_total, int nsets) {
  using namespace updw;
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  const uint32_t sbase = (smem_u32(smem_raw) + 1023u) & ~1023u;
  uint8_t* smem = smem_raw + (sbase - smem_u32(smem_raw));
  uint8_t* ring = smem + W_BYTES;
  float* stg = reinterpret_cast<float*>(ring + STAGES * STAGE_BYTES);
  __shared__ uint64_t tma_full[STAGES], full[STAGES], empty[STAGES], w_full, fwd_full, xbg_free, opnd_ready, opnd_free, grad_done;
  __shared__ uint32_t tmem_base_s;
  __shared__ float loss_red[EPI_WARPS];
  __shared__ float lrmax_s[THREADS / 32];
  __shared__ __align__(16) float ne_s[STAGES][T];   // -eta of the stage's tokens, scaled (0 beyond M)

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int nslices = H / HS;
  const long long U = (long long)nh * nslices * tiles_total;
  const long long lo = blockIdx.x * U / gridDim.x, hi = (blockIdx.x + 1) * U / gridDim.x;
  const int total = (int)(hi - lo);                 // tiles this CTA processes, over all its segments
  // unit lo + gi -> pair (= slice * nh + h) and token tile. Slice-major pairs: when nh divides the
  // CTAs-per-pair pattern (config 5: 4.625 CTAs per pair, nh = 8) the slices of one head walk the
  // same token tiles at the same time, so K / V come from DRAM once and from L2 three times
  auto locate = [&](int gi, int& pair, int& tile) {
    const long long u = lo + gi;
    pair = (int)(u / tiles_total);
    tile = (int)(u - (long long)pair * tiles_total);
  };
  auto load_stage = [&](int gi) {
    int pair, tile;
    locate(gi, pair, tile);
    const int s = gi % STAGES, h = pair % nh, row = tile * T;
    mbar_arrive_expect_tx(&tma_full[s], STAGE_BYTES);
    uint8_t* dst = ring + s * STAGE_BYTES;
    tma_load_2d(dst, &mapK, &tma_full[s], h * HD, row);
    tma_load_2d(dst + SUB_BYTES, &mapK, &tma_full[s], h * HD + 64, row);
    tma_load_2d(dst + TILE_BYTES, &mapV, &tma_full[s], h * HD, row);
    tma_load_2d(dst + TILE_BYTES + SUB_BYTES, &mapV, &tma_full[s], h * HD + 64, row);
  };
  // weights of a pair: mat m (0 = W1^T, 1 = W2, 2 = W3^T), hd half c -> [128 rows x 64] sub-tile
  auto load_weights = [&](int pair) {
    const int h = pair % nh, slice = pair / nh;
    mbar_arrive_expect_tx(&w_full, W_BYTES);
    for (int m = 0; m < 3; ++m)
      for (int c = 0; c < 2; ++c)
        tma_load_2d(smem + m * WMAT_BYTES + c * WSUB_BYTES, &mapW, &w_full, c * 64,
                    (m * nh + h) * H + slice * HS);
  };

  if (tid == 0) {
    for (int s = 0; s < STAGES; ++s) { mbar_init(&tma_full[s], 1); mbar_init(&full[s], CVT_WARPS); mbar_init(&empty[s], 1); }
    mbar_init(&w_full, 1);
    mbar_init(&fwd_full, 1);
    mbar_init(&xbg_free, 1);
    mbar_init(&opnd_ready, EPI_WARPS);
    mbar_init(&opnd_free, 1);
    mbar_init(&grad_done, 1);
    fence_mbar_init();
    tma_prefetch_desc(&mapK);
    tma_prefetch_desc(&mapV);
    tma_prefetch_desc(&mapW);
    if (total > 0) load_weights((int)(lo / tiles_total));
    const int npre = min(total, STAGES);
    for (int gi = 0; gi < npre; ++gi) load_stage(gi);
  }
  __syncwarp();
  // max |eta| over the tokens of all of this CTA's segments (all threads; overlaps the first TMA round trip)
  {
    float mx = 0.f;
    for (long long u = lo; u < hi;) {
      const int pair = (int)(u / tiles_total), t0 = (int)(u - (long long)pair * tiles_total);
      const int n = (int)min(hi - u, (long long)(tiles_total - t0));
      const float* lrh = lr + (size_t)(pair % nh) * M;
      const int t_hi = min(M, (t0 + n) * T);
#pragma unroll 4
      for (int t = t0 * T + tid; t < t_hi; t += THREADS) mx = fmaxf(mx, fabsf(__ldg(lrh + t)));
      u += n;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    if (lane == 0) lrmax_s[warp] = mx;
  }
  if (warp == 0) { tmem_alloc(&tmem_base_s, 512); tmem_relinquish(); }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tb = tmem_base_s;
  if (tb != 0) __trap();      // all 512 columns belong to this CTA: the issuer uses absolute columns
  float eta_sc, eta_isc;      // the gradient operands carry eta * eta_sc; undone at the flush
  {
    float mx = 0.f;
#pragma unroll
    for (int w = 0; w < THREADS / 32; ++w) mx = fmaxf(mx, lrmax_s[w]);
    eta_scale(mx, eta_sc, eta_isc);
  }

  if (warp == 0) {
    // ===================== TMA producer =====================
    if (elect_one()) {
      for (int gi = STAGES; gi < total; ++gi) {      // tiles 0 .. STAGES-1 were requested in the prologue
        mbar_wait(&empty[gi % STAGES], ((gi / STAGES) & 1) ^ 1);
        load_stage(gi);
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer (forward and gradients) =====================
    if (elect_one()) {
      constexpr uint32_t idesc_f = umma_idesc(HS, T, 0, 0, TTT_FMT_F16, TTT_FMT_F16);    // A = weights, B = token tile (fp16), K-major
      constexpr uint32_t idesc_g = umma_idesc(HS, HD, 0, 1, TTT_FMT_F16, TTT_FMT_F16);   // A = fp16 TMEM operand, B = token tile (fp16), MN-major
      const uint64_t dw = umma_smem_desc_sw128(sbase, 16, 1024);
      const uint64_t dr_k = umma_smem_desc_sw128(sbase + W_BYTES, 16, 1024);
      const uint64_t dr_mn = umma_smem_desc_sw128(sbase + W_BYTES, SUB_BYTES, 1024);   // 2nd hd atom: +SUB_BYTES
      // forward product of weight matrix m with the K (tile_off 0) or V tile of stage offset st
      auto forward = [&](int m, uint64_t st, uint32_t dcol) {
#pragma unroll
        for (int k = 0; k < HD / 16; ++k) {
          const uint64_t a = dw + (uint64_t)(m * (WMAT_BYTES >> 4) + (k >> 2) * (WSUB_BYTES >> 4) + (k & 3) * 2);
          const uint64_t b = dr_k + st + (uint64_t)((k >> 2) * (SUB_BYTES >> 4) + (k & 3) * 2);
          umma_ss(dcol, a, b, idesc_f, k > 0);
        }
      };
      // gradient MMAs of a tile, in two groups: G2 reads Hd' from the x columns and must precede the next
      // x product; G1 / G3 read their own operand columns and fill the pipe while the epilogue loads x | b | g
      auto grad_w2 = [&](uint64_t st, uint32_t acc) {
#pragma unroll
        for (int k = 0; k < T / 16; ++k)                     // +2048 B per 16-token K step
          umma_ts(C_G2, C_OH + 8 * k, dr_mn + st + (TILE_BYTES >> 4) + 128 * k, idesc_g, acc | k);
      };
      auto grad_w13 = [&](uint64_t st, uint32_t acc) {
#pragma unroll
        for (int k = 0; k < T / 16; ++k) {
          umma_ts(C_G1, C_OA + 8 * k, dr_mn + st + 128 * k, idesc_g, acc | k);
          umma_ts(C_G3, C_OB + 8 * k, dr_mn + st + 128 * k, idesc_g, acc | k);
        }
      };
      int gi = 0, seg = 0;
      while (gi < total) {
        int pair, t0;
        locate(gi, pair, t0);
        const int n = min(total - gi, tiles_total - t0);     // tiles of this segment
        if (seg > 0) {                 // every MMA that read the previous pair's weights has completed
          mbar_wait(&grad_done, (seg - 1) & 1);
          load_weights(pair);
        }
        mbar_wait(&w_full, seg & 1);
        uint64_t st_prev = 0;
        int s_prev = 0;
        for (int i = 0; i < n; ++i, ++gi) {
          const int s = gi % STAGES;
          const uint64_t st = (uint64_t)s * (STAGE_BYTES >> 4);
          mbar_wait(&full[s], (gi / STAGES) & 1);
          if (i > 0) mbar_wait(&xbg_free, (gi - 1) & 1);       // x | b | g of the previous tile are in registers
          tc_fence_after();
          forward(2, st, C_B);
          forward(1, st + (TILE_BYTES >> 4), C_G);
          if (i > 0) {
            mbar_wait(&opnd_ready, (gi - 1) & 1);
            tc_fence_after();
            grad_w2(st_prev, i > 1);
          }
          forward(0, st, C_X);           // after the gradient MMAs that read Hd' from these columns
          tc_commit(&fwd_full);
          if (i > 0) {
            grad_w13(st_prev, i > 1);    // runs while the epilogue of tile i loads its accumulators
            tc_commit(&opnd_free);       // 2 dA | dB operand columns may be overwritten
            tc_commit(&empty[s_prev]);
          }
          st_prev = st;
          s_prev = s;
        }
        mbar_wait(&opnd_ready, (gi - 1) & 1);
        tc_fence_after();
        grad_w2(st_prev, n > 1);
        grad_w13(st_prev, n > 1);
        tc_commit(&opnd_free);
        tc_commit(&empty[s_prev]);
        tc_commit(&grad_done);
        ++seg;
      }
    }
  } else if (warp == 2) {
    // ===================== stage finisher 0: fp16 conversion, learning rates =====================
    // When the TMA has landed a stage, the CVT_WARPS finisher warps convert its K and V tiles from bf16
    // to fp16 in place, a quarter of the 16 KB each (all MMA operands are fp16, ttt_internal.h), and this
    // one also puts -eta of the tile's 32 tokens (one 128-B line of lr, scaled by the CTA's power of
    // two) into the stage's slot; the global loads of lr run LRPF tiles ahead of the ring (register
    // double buffer)
    constexpr int LRPF = 4;
    auto ld_batch = [&](int g0, float (&v)[LRPF]) {
#pragma unroll
      for (int u = 0; u < LRPF; ++u) {
        float x = 0.f;
        if (g0 + u < total) {
          int pair, tile;
          locate(g0 + u, pair, tile);
          const int t = tile * T + lane;
          if (t < M) x = -eta_sc * __ldg(lr + (size_t)(pair % nh) * M + t);
        }
        v[u] = x;
      }
    };
    float cur[LRPF], nxt[LRPF];
    ld_batch(0, cur);
    for (int g0 = 0; g0 < total; g0 += LRPF) {
      ld_batch(g0 + LRPF, nxt);
#pragma unroll
      for (int u = 0; u < LRPF; ++u) {
        const int gi = g0 + u;
        if (gi < total) {
          const int s = gi % STAGES, it = gi / STAGES;
          mbar_wait(&tma_full[s], it & 1);       // (the TMA was issued after the stage's `empty`)
          tile_bf16_to_f16<STAGE_BYTES / 512 / CVT_WARPS>(ring + s * STAGE_BYTES, lane);
          ne_s[s][lane] = cur[u];
          fence_proxy_async_smem();
          __syncwarp();
          if (lane == 0) mbar_arrive(&full[s]);
        }
      }
#pragma unroll
      for (int u = 0; u < LRPF; ++u) cur[u] = nxt[u];
    }
  } else if (warp == 3 || warp >= 4 + EPI_WARPS) {
    // ===================== stage finishers 1 .. CVT_WARPS-1: fp16 conversion =====================
    const int part = warp == 3 ? 1 : warp - (4 + EPI_WARPS) + 2;
    for (int gi = 0; gi < total; ++gi) {
      const int s = gi % STAGES;
      mbar_wait(&tma_full[s], (gi / STAGES) & 1);
      tile_bf16_to_f16<STAGE_BYTES / 512 / CVT_WARPS>(ring + s * STAGE_BYTES + part * (STAGE_BYTES / CVT_WARPS), lane);
      fence_proxy_async_smem();
      __syncwarp();
      if (lane == 0) mbar_arrive(&full[s]);
    }
  } else if (warp >= 4) {
    // ===================== epilogue warps =====================
    const int ew = warp - 4, q = warp & 3, kh = ew >> 2;   // lane quadrant, K step (16 tokens) of the tile
    const int j = q * 32 + lane;                           // hidden unit within the slice = TMEM lane
    const uint32_t lane_base = static_cast<uint32_t>(q * 32) << 16;
    const uint64_t ONE2 = pack2(1.0f, 1.0f), NONE2 = pack2(-1.0f, -1.0f), HALF2 = pack2(0.5f, 0.5f);
    const size_t me = (size_t)nh * H * HD;
    int gi = 0, seg = 0;
    while (gi < total) {
      int pair, t0;
      locate(gi, pair, t0);
      const int n = min(total - gi, tiles_total - t0);
      uint64_t loss2 = 0ull;
      for (int i = 0; i < n; ++i, ++gi) {
        const int s = gi % STAGES;
        mbar_wait(&fwd_full, gi & 1);
        mbar_wait(&full[s], (gi / STAGES) & 1);              // acquire of the loader's -eta slot
        tc_fence_after();
        const uint2* nes = reinterpret_cast<const uint2*>(&ne_s[s][16 * kh]);
        uint32_t rx[16], rb[16], rg[16];
        tmem_ld_x16(lane_base + C_X + 16 * kh, rx);
        tmem_ld_x16(lane_base + C_B + 16 * kh, rb);
        tmem_ld_x16(lane_base + C_G + 16 * kh, rg);
        tc_wait_ld();
        tc_fence_before();
        asm volatile("bar.sync 1, 256;" ::: "memory");       // every warp holds its x | b | g
        if (ew == 0 && lane == 0) mbar_arrive(&xbg_free);
        uint32_t pa[8], pb[8], ph[8];
#pragma unroll
        for (int c = 0; c < 16; c += 2) {
          const uint64_t x = fmul2(pack2u(rx[c], rx[c + 1]), HALF2);   // a / 2
          const uint64_t bb = pack2u(rb[c], rb[c + 1]);
          const uint2 nev = nes[c >> 1];
          const uint64_t ne = pack2u(nev.x, nev.y);
          const uint64_t g = fmul2(ne, pack2u(rg[c], rg[c + 1]));   // dHd = (-eta v) W2^T
          float x0, x1;
          unpack2(x, x0, x1);
          const uint64_t th = pack2(tanh_approx(x0), tanh_approx(x1));
          const uint64_t S = ffma2(x, th, x);                  // SiLU(a) = a sigmoid(a), a = 2 x
          const uint64_t p = fadd2(th, ONE2);                  // 2 sigmoid(a)
          const uint64_t m = ffma2(th, NONE2, ONE2);           // 2 (1 - sigmoid(a))
          const uint64_t t2 = ffma2(S, m, p);                  // 2 SiLU'(a)
          const uint64_t hdv = fmul2(S, bb);                   // hidden activation Hd
          pa[c >> 1] = pack_f16x2_from2(fmul2(fmul2(g, bb), t2));   // 2 dA
          pb[c >> 1] = pack_f16x2_from2(fmul2(g, S));               // dB
          ph[c >> 1] = pack_f16x2_from2(fmul2(ne, hdv));            // Hd' = -eta Hd
          if (LOSS) loss2 = ffma2(hdv, g, loss2);
        }
        // Hd' columns: their last readers (W2-gradient MMAs of the previous tile) were issued before the x
        // MMAs of this tile and are covered by fwd_full; 2 dA | dB columns: released by the commit after
        // the W1 / W3 gradient MMAs of the previous tile
        if (gi > 0) { mbar_wait(&opnd_free, (gi - 1) & 1); tc_fence_after(); }
        tmem_st_x8(lane_base + C_OA + 8 * kh, pa);
        tmem_st_x8(lane_base + C_OB + 8 * kh, pb);
        tmem_st_x8(lane_base + C_OH + 8 * kh, ph);
        tc_wait_st();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(&opnd_ready);
      }
      // a dependent kernel (PDL) may be scheduled from here on; it still waits for this grid to finish
      if (gi >= total) asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
      // ---- flush the segment's gradient accumulators: one fp32 partial slice ----
      mbar_wait(&grad_done, seg & 1);
      tc_fence_after();
      const int h = pair % nh, slice = pair / nh;
      // ordinal of this segment within its pair = this CTA's index among the CTAs that touch the pair
      int ord;
      {
        const long long target = (long long)pair * tiles_total, n_cta = gridDim.x;
        long long c1 = target * n_cta / U;
        while (c1 > 0 && (c1 * U) / n_cta > target) --c1;
        while (((c1 + 1) * U) / n_cta <= target) ++c1;
        ord = (int)(blockIdx.x - c1);
      }
      const bool pair_done = t0 + n == tiles_total;          // zero-fill the sets no segment writes
      // TMEM gives a thread columns of ONE row; stored directly, a warp store would touch 32 lines for
      // 512 bytes. Each 64-column half of a matrix is staged as [128][68] fp32 in shared memory and
      // leaves as full lines (the slice's rows are contiguous in the partial set).
      const size_t slice_base = ((size_t)h * H + (size_t)slice * HS) * HD;
      const uint32_t gcol[3] = {C_G1, C_G2, C_G3};
      const int et = ew * 32 + lane;                         // 0 .. 255
#pragma unroll
      for (int mat = 0; mat < 3; ++mat) {
        const float sc = (mat == 0 ? 0.5f : 1.0f) * eta_isc; // G1 was accumulated from 2 dA; eta scale undone
#pragma unroll
        for (int p = 0; p < 2; ++p) {                        // column half; its four warps fill the stage
          if (kh == p) {
#pragma unroll
            for (int cc = 0; cc < 4; ++cc) {
              uint32_t r[16];
              tmem_ld_x16(lane_base + gcol[mat] + 64 * p + 16 * cc, r);
              tc_wait_ld();
              float4* d = reinterpret_cast<float4*>(stg + j * SLD + 16 * cc);
#pragma unroll
              for (int v = 0; v < 4; ++v)
                d[v] = make_float4(sc * __uint_as_float(r[4 * v]), sc * __uint_as_float(r[4 * v + 1]),
                                   sc * __uint_as_float(r[4 * v + 2]), sc * __uint_as_float(r[4 * v + 3]));
            }
          }
          asm volatile("bar.sync 1, 256;" ::: "memory");
          const size_t e0 = mat * me + slice_base + 64 * p;
#pragma unroll
          for (int k = 0; k < HS * 64 / 4 / 256; ++k) {
            const int e = et + 256 * k, rr = e >> 4, c4 = e & 15;   // row, float4 within the 64-column half
            const size_t g = e0 + (size_t)rr * HD + 4 * c4;
            *reinterpret_cast<float4*>(P + (size_t)ord * 3 * me + g) =
                *reinterpret_cast<const float4*>(stg + rr * SLD + 4 * c4);
            if (pair_done)
              for (int z = ord + 1; z < nsets; ++z)
                *reinterpret_cast<float4*>(P + (size_t)z * 3 * me + g) = make_float4(0.f, 0.f, 0.f, 0.f);
          }
          asm volatile("bar.sync 1, 256;" ::: "memory");
        }
      }
      tc_fence_before();
      if (LOSS) {
        float l0, l1;
        unpack2(loss2, l0, l1);
        float loss = l0 + l1;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) loss += __shfl_xor_sync(0xffffffffu, loss, o);
        if (lane == 0) loss_red[ew] = loss;
        asm volatile("bar.sync 1, 256;" ::: "memory");
        if (ew == 0 && lane == 0) {
          float t = 0.f;
          for (int w = 0; w < EPI_WARPS; ++w) t += loss_red[w];
          loss_part[((size_t)ord * nslices + slice) * nh + h] = t * eta_isc;
          if (pair_done)
            for (int z = ord + 1; z < nsets; ++z) loss_part[((size_t)z * nslices + slice) * nh + h] = 0.f;
        }
        asm volatile("bar.sync 1, 256;" ::: "memory");
      }
      ++seg;
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 0) tmem_dealloc(tb, 512);
}

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------
int bf16_update_wide_supported(const ttt_config* cfg) {
  return cfg->hd == updw::HD && cfg->hidden % updw::HS == 0 && !cfg->linear_fast_weight;
}

// CTAs of the launch and partial sets it writes: units = pairs x tiles spread evenly over the SMs;
// nsets = the largest number of CTAs whose range touches one (head, slice) pair
static void wide_geometry(const ttt_ctx* ctx, int64_t M, int* tiles, int* ncta, int* nsets) {
  const int t = (int)((M + updw::T - 1) / updw::T);
  const int pairs = ctx->cfg.nh * (ctx->cfg.hidden / updw::HS);
  const long long U = (long long)pairs * t;
  int n = ctx->sm_count;
  if (n > U) n = (int)U;
  if (n < 1) n = 1;
  int worst = 1;
  for (int p = 0; p < pairs && U > 0; ++p) {
    // first CTA with hi(c) > p t, last CTA with lo(c) < (p + 1) t
    long long c0 = (long long)p * t * n / U;
    while (c0 > 0 && (c0 * U) / n > (long long)p * t) --c0;
    while (((c0 + 1) * U) / n <= (long long)p * t) ++c0;
    long long c1 = c0;
    while (c1 + 1 < n && ((c1 + 1) * U) / n < (long long)(p + 1) * t) ++c1;
    if ((int)(c1 - c0 + 1) > worst) worst = (int)(c1 - c0 + 1);
  }
  *tiles = t;
  *ncta = n;
  *nsets = worst;
}

int bf16_wide_partials_needed(const ttt_ctx* ctx, int64_t M) {
  int t, n, s;
  wide_geometry(ctx, M, &t, &n, &s);
  return s;
}

// appends `*used` partial-gradient sets, `*loss_rows` loss partial rows
int bf16_accumulate_wide(ttt_ctx* ctx, const __nv_bfloat16* K, const __nv_bfloat16* V, const float* lr,
                         int64_t M, int64_t ld, bool want_loss, int* used, int* loss_rows,
                         cudaStream_t s) {
  const ttt_config& c = ctx->cfg;
  int tiles, ncta, nsets;
  wide_geometry(ctx, M, &tiles, &ncta, &nsets);
  CUtensorMap mapK, mapV, mapW;
  int rc = make_token_map(ctx, &mapK, K, M, (int64_t)c.nh * c.hd, ld, updw::T);
  if (rc != TTT_OK) return rc;
  rc = make_token_map(ctx, &mapV, V, M, (int64_t)c.nh * c.hd, ld, updw::T);
  if (rc != TTT_OK) return rc;
  // fp16 operand copy of the weights as one [3 nh H][hd] matrix, boxes of [128 rows][64]
  rc = make_token_map(ctx, &mapW, ctx->Wb, (int64_t)3 * c.nh * c.hidden, c.hd, c.hd, updw::HS);
  if (rc != TTT_OK) return rc;
  if (!(ctx->attr_done & ATTR_UPDW)) {
    TTT_CUDA_TRY(ctx, cudaFuncSetAttribute(bf16_update_wide_kernel<false>,
                                           cudaFuncAttributeMaxDynamicSharedMemorySize,
                                           (int)updw::SMEM_BYTES), "bf16_update_wide_kernel smem attr");
    TTT_CUDA_TRY(ctx, cudaFuncSetAttribute(bf16_update_wide_kernel<true>,
                                           cudaFuncAttributeMaxDynamicSharedMemorySize,
                                           (int)updw::SMEM_BYTES), "bf16_update_wide_kernel smem attr");
    ctx->attr_done |= ATTR_UPDW;
  }
  float* P = ctx->partials + (size_t)ctx->n_partials * 3 * ctx->mat_elems;
  if (want_loss)
    bf16_update_wide_kernel<true><<<ncta, updw::THREADS, updw::SMEM_BYTES, s>>>(
        mapK, mapV, mapW, lr, P, ctx->loss_part, (int)M, c.nh, c.hidden, tiles, nsets);
  else
    bf16_update_wide_kernel<false><<<ncta, updw::THREADS, updw::SMEM_BYTES, s>>>(
        mapK, mapV, mapW, lr, P, ctx->loss_part, (int)M, c.nh, c.hidden, tiles, nsets);
  TTT_LAUNCH_CHECK(ctx, "bf16_update_wide_kernel");
  *used = nsets;
  *loss_rows = nsets * (c.hidden / updw::HS);
  return TTT_OK;
}

}  // namespace ttt
