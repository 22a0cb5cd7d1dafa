// bf16_apply_wide_pair.cu — the hd = 128 apply kernel (O = (SiLU(Q W1) * (Q W3)) W2, Eq. 4 with
// Eq. 12, weights streamed from L2) on CTA PAIRS: tcgen05.mma.cta_group::2, M = 256.
//
// Why pairs: with M = 128 the B-operand reads of an N = 128 MMA alone need the full 128 B/clk of the
// shared-memory port at the nominal tensor rate, and the streamed weights add their TMA writes on
// top (a single-CTA version of this kernel measured ~112 clk per M128 N128 K16 MMA against a floor of 64).
// A CTA pair shares every B operand: each CTA streams and reads HALF of a step's weights —
//   forward   x | b [256 x 128] = Q [256 x 128] . [W1^T rows ; W3^T rows]^T : rank 0 holds the 64 W1^T
//             rows (N 0-63 = x), rank 1 the 64 W3^T rows (N 64-127 = b) of the 64-hidden step;
//   down      O [256 x 128] += Hq [256 x 64] . W2 rows [64 x 128]: rank r holds hd columns 64 r .. 64 r + 63
// — while its 128 token rows of A (Q in shared memory, Hq in TMEM) and of the accumulators stay in
// its own SM. Rank 0 issues every MMA; commits are multicast to both CTAs' barriers; the TMA loads of
// both CTAs complete on rank 0's barriers; rank 1's warps arrive on rank 0's barriers remotely.
//
// Pipeline: with the MMAs at their floor the F -> SwiGLU epilogue -> D chain of a token tile is what
// limits a step (first pair version, two tiles per CTA with single forward buffers as in the
// single-CTA kernel: 177 us at cfg5 — both tiles' epilogues ran in lock-step, 2 000 of 3 650 clk per
// step the issuer waited for Hq). So a unit is (head, ONE 128-token tile per CTA = 256 tokens per pair),
// the forward accumulators x | b are triple-buffered (F(g + 3) follows the completion of D(g)), all
// 16 epilogue warps work on the one tile, and eight warps of their own drain the O accumulator to
// global memory. TMEM (512 columns): O at 0, x | b [3] at 128 / 256 / 384 (64 + 64 columns); the bf16
// Hq (A operand of the down MMAs) overwrites the first 32 columns of its own x once all epilogue
// warps hold their x | b in registers.
#include <stdio.h>

#include "tc_common.cuh"
#include "ttt_internal.h"

namespace ttt {

int make_token_map(ttt_ctx* ctx, CUtensorMap* map, const void* base, int64_t rows, int64_t cols,
                   int64_t ld, int box_rows);   // bf16_update.cu

namespace appp {
constexpr int HD = 128;        // head dimension
constexpr int TM = 128;        // tokens per tile and CTA (MMA M = 256 over the pair)
constexpr int HSTEP = 64;      // hidden units per step
constexpr int NST = 4;         // weight ring stages (24 KB per CTA and stage)
constexpr int EPI_WARPS = 16;  // SwiGLU epilogue warps (4 per TMEM lane quadrant, 16 hidden columns each)
constexpr int DRAIN_WARPS = 8; // O -> bf16 -> global (2 per TMEM lane quadrant, 64 columns each)
constexpr int DRAIN_WARP0 = 4 + EPI_WARPS;
constexpr int THREADS = (4 + EPI_WARPS + DRAIN_WARPS) * 32;
constexpr int QSUB_BYTES = TM * 128;            // [128 tokens x 64] bf16 sub-tile (half of hd)
constexpr int QTILE_BYTES = 2 * QSUB_BYTES;
constexpr int BOX_BYTES = HSTEP * 128;          // one TMA box of weights: [64 rows x 64]
constexpr int W2_OFF = 2 * BOX_BYTES;           // after the two hd halves of this CTA's forward rows
constexpr int WSTAGE_BYTES = 3 * BOX_BYTES;     // per CTA
constexpr size_t SMEM_BYTES = 2 * (size_t)QTILE_BYTES + (size_t)NST * WSTAGE_BYTES + 1024;
constexpr int NF = 3;          // forward accumulator buffers x | b (128 columns each)
constexpr uint32_t C_O = 0, C_F = 128;
}  // namespace appp

__global__ void __launch_bounds__(appp::THREADS, 1)
bf16_apply_wide_pair_kernel(const __grid_constant__ CUtensorMap mapW, const __grid_constant__ CUtensorMap mapQ,
                            __nv_bfloat16* __restrict__ O, int M, int64_t ld, int nh, int H, int npairs,
                            int q_early) {
  using namespace appp;
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  const uint32_t sbase = (smem_u32(smem_raw) + 1023u) & ~1023u;
  uint8_t* smem = smem_raw + (sbase - smem_u32(smem_raw));
  uint8_t* wring = smem + 2 * QTILE_BYTES;
  // Slot k-th use: "full"-type barriers are waited with parity k & 1, "free"-type ones (before the
  // k-th use, k >= 1) with (k - 1) & 1. w_full, q_full, hq_ready, o_free are waited on by rank 0 only
  // (its copies collect both CTAs).
  __shared__ uint64_t w_full[NST], w_empty[NST], q_full[2], q_free[2], f_full[NF], hq_ready[NF],
      o_full, o_free;
  __shared__ uint32_t tmem_base_s;

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const uint32_t rank = cluster_rank();
  const int nstep = H / HSTEP;
  const int nunits = nh * npairs;
  const int cid = blockIdx.x >> 1, ncl = gridDim.x >> 1;
  const int my_units = cid < nunits ? (nunits - cid + ncl - 1) / ncl : 0;
  const int G = my_units * nstep;                // steps of this pair, all units

  if (tid == 0) {
    for (int s = 0; s < NST; ++s) { mbar_init(&w_full[s], 1); mbar_init(&w_empty[s], 1); }
    for (int b = 0; b < 2; ++b) { mbar_init(&q_full[b], 1); mbar_init(&q_free[b], 1); }
    for (int b = 0; b < NF; ++b) { mbar_init(&f_full[b], 1); mbar_init(&hq_ready[b], 2 * EPI_WARPS); }
    mbar_init(&o_full, 1);
    mbar_init(&o_free, 2 * DRAIN_WARPS);
    fence_mbar_init();
    tma_prefetch_desc(&mapW);
    tma_prefetch_desc(&mapQ);
  }
  __syncthreads();
  cluster_sync_all();            // the peer's barriers exist before anything can arrive on them
  if (warp == 0) { tmem_alloc2(&tmem_base_s, 512); tmem_relinquish2(); }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tb = tmem_base_s;
  if (tb != 0) __trap();      // all 512 columns belong to this pair: absolute columns below
  // Q of a unit: this CTA's tile into Q buffer `qb`, completion on rank 0's barrier
  auto load_q = [&](int unit, int qb) {
    const int h = unit / npairs, p = unit % npairs;
    if (rank == 0) mbar_arrive_expect_tx(&q_full[qb], 2 * QTILE_BYTES);
    const uint32_t qbar = mapa_u32(&q_full[qb], 0);
    for (int c = 0; c < 2; ++c)
      tma_load_2d_pair(smem + qb * QTILE_BYTES + c * QSUB_BYTES, &mapQ, qbar, h * HD + c * 64,
                       (2 * p + (int)rank) * TM);
  };
  // inside ttt_chunk_step (the kernels ahead in the stream are the library's own and do not write Q)
  // the first unit's Q is requested before the dependency wait
  if (q_early && tid == 0 && my_units > 0) load_q(cid, 0);
  // programmatic dependent launch: everything above overlapped the tail of the commit kernel
  asm volatile("griddepcontrol.wait;" ::: "memory");

  if (warp == 0) {
    // ===================== TMA producer (both CTAs; completion on rank 0's barriers) =====================
    if (elect_one()) {
      int g = 0;
      for (int u = 0; u < my_units; ++u) {
        const int unit = cid + u * ncl, h = unit / npairs;
        const int qb = u & 1;
        if (u >= 2) mbar_wait(&q_free[qb], ((u >> 1) - 1) & 1);   // the forward MMAs of unit u - 2 are done
        if (u > 0 || !q_early) load_q(unit, qb);
        for (int n = 0; n < nstep; ++n, ++g) {
          const int s = g % NST;
          if (g >= NST) mbar_wait(&w_empty[s], ((g / NST) - 1) & 1);
          if (rank == 0) mbar_arrive_expect_tx(&w_full[s], 2 * WSTAGE_BYTES);
          const uint32_t bar = mapa_u32(&w_full[s], 0);
          uint8_t* dst = wring + s * WSTAGE_BYTES;
          const int rf = ((rank ? 2 : 0) * nh + h) * H + n * HSTEP;     // W1^T rows (rank 0) / W3^T rows (rank 1)
          const int r2 = (1 * nh + h) * H + n * HSTEP;
          tma_load_2d_pair(dst, &mapW, bar, 0, rf);
          tma_load_2d_pair(dst + BOX_BYTES, &mapW, bar, 64, rf);
          tma_load_2d_pair(dst + W2_OFF, &mapW, bar, 64 * (int)rank, r2);
        }
      }
    }
  } else if (warp == 1) {
    // ===================== forward-MMA issuer (rank 0 only) =====================
    // Two issuing threads (this one and warp 2): an MMA issue costs its thread ~45 clk, a multicast
    // commit ~200, a barrier probe ~90 — one thread issuing a step's 12 MMAs and 2-3 commits needs
    // ~1 000 clk against 768 clk of tensor work.
    if (rank == 0 && elect_one() && G > 0) {
      constexpr uint32_t idesc_f = umma_idesc(2 * TM, 2 * HSTEP, 0, 0, TTT_FMT_BF16, TTT_FMT_BF16);   // A = Q (smem), B = forward rows, K-major
      const uint64_t dq = umma_smem_desc_sw128(sbase, 16, 1024);
      const uint64_t dwf = umma_smem_desc_sw128(sbase + 2 * QTILE_BYTES, 16, 1024);
      // x | b of step g <- Q(unit) [W1^T | W3^T]^T of the step's ring stage. F(g) overwrites the
      // x | b (and Hq) of step g - NF: it waits until D(g - NF) has completed (= its stage is free).
      int n = 0, qb = 0, st = 0, fb = 0, sw = 0;
      uint32_t qph = 0, sph = 0, swph = 0;
      for (int g = 0; g < G; ++g) {
        // operands first (they landed long ago), the buffer's release by D(g - NF) last: that wait is
        // on the critical cycle F -> epilogue -> D -> F, the others are not. Polling waits: a
        // suspended try_wait wakes ~230 clk after the phase completes.
        if (n == 0) mbar_wait(&q_full[qb], qph);
        mbar_wait(&w_full[st], sph);
        if (g >= NF) {
          mbar_wait_spin(&w_empty[sw], swph);
          if (++sw == NST) { sw = 0; swph ^= 1; }
        }
        tc_fence_after();
        const uint64_t a0 = dq + (uint64_t)(qb * (QTILE_BYTES >> 4));
        const uint64_t b0 = dwf + (uint64_t)(st * (WSTAGE_BYTES >> 4));
        const uint32_t acc = C_F + fb * 128;
#pragma unroll
        for (int k = 0; k < HD / 16; ++k)
          umma_ss2(acc, a0 + (uint64_t)((k >> 2) * (QSUB_BYTES >> 4) + (k & 3) * 2),
                   b0 + (uint64_t)((k >> 2) * (BOX_BYTES >> 4) + (k & 3) * 2), idesc_f, k > 0);
        tc_commit2(&f_full[fb]);
        if (++n == nstep) { tc_commit2(&q_free[qb]); n = 0; if (qb) qph ^= 1; qb ^= 1; }
        if (++st == NST) { st = 0; sph ^= 1; }
        if (++fb == NF) fb = 0;
      }
    }
  } else if (warp == 2) {
    // ===================== down-MMA issuer (rank 0 only) =====================
    if (rank == 0 && elect_one() && G > 0) {
      constexpr uint32_t idesc_d = umma_idesc(2 * TM, HD, 0, 1, TTT_FMT_BF16, TTT_FMT_BF16);          // A = Hq (TMEM), B = W2 rows, MN-major
      const uint64_t dw2 = umma_smem_desc_sw128(sbase + 2 * QTILE_BYTES + W2_OFF, BOX_BYTES, 1024);
      // O(unit) (+)= Hq(step g) W2[step rows]; the step's W2 rows landed with its forward rows
      // (w_full was waited on by the forward issuer before F(g), which precedes Hq(g))
      int n = 0, u = 0, st = 0, fb = 0;
      uint32_t fph = 0;
      for (int g = 0; g < G; ++g) {
        if (n == 0 && u > 0) mbar_wait_spin(&o_free, (u - 1) & 1);   // O of the previous unit has been read
        mbar_wait_spin(&hq_ready[fb], fph);
        tc_fence_after();
        const uint64_t b0 = dw2 + (uint64_t)(st * (WSTAGE_BYTES >> 4));
        const uint32_t hq = C_F + fb * 128;
#pragma unroll
        for (int k = 0; k < HSTEP / 16; ++k)             // +2048 B per 16 hidden rows
          umma_ts2(C_O, hq + 8 * k, b0 + 128 * k, idesc_d, (n > 0) | k);
        tc_commit2(&w_empty[st]);
        if (++n == nstep) { tc_commit2(&o_full); n = 0; ++u; }
        if (++st == NST) st = 0;
        if (++fb == NF) { fb = 0; fph ^= 1; }
      }
    }
  } else if (warp >= 4 && warp < DRAIN_WARP0) {
    // ===================== SwiGLU epilogue warps =====================
    // All 16 warps work on every step (4 per TMEM lane quadrant, 16 hidden columns each): the
    // epilogue is on the critical cycle F -> epilogue -> D -> F, so its latency counts, not its
    // throughput (two groups of 8 warps alternating steps share the MUFU pipe and take 1 350 clk per
    // step each against 900 for the step handled by all warps).
    const int ew = warp - 4, q = warp & 3, cg = ew >> 2;   // lane quadrant, 16-column group of the step's 64
    const uint32_t lane_base = static_cast<uint32_t>(q * 32) << 16;
    const uint64_t HALF2 = pack2(0.5f, 0.5f);
    int fb = 0;
    uint32_t fph = 0;
    for (int g = 0; g < G; ++g) {
      const uint32_t buf = lane_base + C_F + fb * 128;
      mbar_wait(&f_full[fb], fph);
      tc_fence_after();
      uint32_t rx[16], rb[16];
      tmem_ld_x16(buf + 16 * cg, rx);
      tmem_ld_x16(buf + 64 + 16 * cg, rb);
      tc_wait_ld();
      tc_fence_before();
      // every epilogue warp holds its x | b: x may be overwritten by Hq (named barrier 1, 16 warps)
      asm volatile("bar.sync 1, 512;" ::: "memory");
      uint32_t ph[8];
#pragma unroll
      for (int c = 0; c < 16; c += 2) {
        const uint64_t x = fmul2(pack2u(rx[c], rx[c + 1]), HALF2);   // a / 2
        float x0, x1;
        unpack2(x, x0, x1);
        const uint64_t th = pack2(tanh_approx(x0), tanh_approx(x1));
        const uint64_t S = ffma2(x, th, x);                          // SiLU(a) = a/2 (1 + tanh(a/2))
        ph[c >> 1] = pack_bf16x2_from2(fmul2(S, pack2u(rb[c], rb[c + 1])));
      }
      tmem_st_x8(buf + 8 * cg, ph);
      tc_wait_st();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) {
        if (rank == 0) mbar_arrive(&hq_ready[fb]); else mbar_arrive_remote(&hq_ready[fb], 0);
      }
      if (++fb == NF) { fb = 0; fph ^= 1; }
    }
  } else if (warp >= DRAIN_WARP0) {
    // ===================== O drain warps: O(unit) -> bf16 -> global =====================
    const int q = warp & 3, half = (warp - DRAIN_WARP0) >> 2;
    const uint32_t lane_base = static_cast<uint32_t>(q * 32) << 16;
    const int row = q * 32 + lane;                         // token row of the tile = TMEM lane
    for (int u = 0; u < my_units; ++u) {
      const int unit = cid + u * ncl, h = unit / npairs, p = unit % npairs;
      mbar_wait(&o_full, u & 1);
      tc_fence_after();
      const int64_t tok = (int64_t)(2 * p + (int)rank) * TM + row;
      // this thread's 64 columns are pulled into registers (packed to bf16 on the fly) before the
      // first store: the single O accumulator is released after two TMEM round trips — the drain
      // sits between the last D of a unit and the first D of the next
      uint32_t pk[32];
#pragma unroll
      for (int part = 0; part < 2; ++part) {               // 32 columns per TMEM round trip
        uint32_t ro[32];
        tmem_ld_x32(lane_base + C_O + 64 * half + 32 * part, ro);
        tc_wait_ld();
#pragma unroll
        for (int v = 0; v < 16; ++v)
          pk[16 * part + v] = pack_bf16x2(__uint_as_float(ro[2 * v]), __uint_as_float(ro[2 * v + 1]));
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) {
        if (rank == 0) mbar_arrive(&o_free); else mbar_arrive_remote(&o_free, 0);
      }
      if (tok < M) {
        uint4* dst = reinterpret_cast<uint4*>(O + tok * ld + h * HD + 64 * half);
#pragma unroll
        for (int v = 0; v < 8; ++v) dst[v] = make_uint4(pk[4 * v], pk[4 * v + 1], pk[4 * v + 2], pk[4 * v + 3]);
      }
    }
  }
  // neither CTA may leave (or free TMEM) while the pair's MMAs, remote arrivals or multicast commits
  // can still touch it
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();
  if (warp == 0) tmem_dealloc2(tb, 512);
}

// ------------------------------------------------------------------------------------------------
int bf16_apply_wide_supported(const ttt_config* cfg) {
  return cfg->hd == appp::HD && cfg->hidden % appp::HSTEP == 0 && !cfg->linear_fast_weight;
}

int bf16_apply_wide_pair(ttt_ctx* ctx, const __nv_bfloat16* Q, __nv_bfloat16* O, int64_t M, int64_t ld,
                         cudaStream_t s) {
  const ttt_config& c = ctx->cfg;
  const int tiles = (int)((M + appp::TM - 1) / appp::TM);
  const int npairs = (tiles + 1) / 2;
  CUtensorMap mapW, mapQ;
  int rc = make_token_map(ctx, &mapW, ctx->Wq, (int64_t)3 * c.nh * c.hidden, c.hd, c.hd, appp::HSTEP);
  if (rc != TTT_OK) return rc;
  rc = make_token_map(ctx, &mapQ, Q, M, (int64_t)c.nh * c.hd, ld, appp::TM);
  if (rc != TTT_OK) return rc;
  if (!(ctx->attr_done & ATTR_APPW)) {
    TTT_CUDA_TRY(ctx, cudaFuncSetAttribute(bf16_apply_wide_pair_kernel,
                                           cudaFuncAttributeMaxDynamicSharedMemorySize,
                                           (int)appp::SMEM_BYTES), "bf16_apply_wide_pair_kernel smem attr");
    ctx->attr_done |= ATTR_APPW;
  }
  cudaLaunchConfig_t cfg = {};
  cfg.blockDim = dim3(appp::THREADS);
  cfg.dynamicSmemBytes = appp::SMEM_BYTES;
  cfg.stream = s;
  cudaLaunchAttribute attr[2];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = 2;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[1].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  // persistent CTA pairs, units round-robin: one wave only — a pair that had to wait for a free
  // TPC would start when the others are done (not every SM of the device can host a pair)
  if (ctx->max_pairs == 0) {
    cfg.gridDim = dim3(2 * (ctx->sm_count / 2));
    int n = 0;
    TTT_CUDA_TRY(ctx, cudaOccupancyMaxActiveClusters(&n, bf16_apply_wide_pair_kernel, &cfg),
                 "bf16_apply_wide_pair_kernel occupancy");
    ctx->max_pairs = n > 0 ? n : -1;
  }
  if (ctx->max_pairs < 0)
    return set_error(ctx, TTT_ERR_UNSUPPORTED, "hd = 128 apply: this device cannot host a CTA pair "
                     "(cta_group::2) of bf16_apply_wide_pair_kernel", cudaSuccess);
  cfg.numAttrs = 2;
  int ncl = c.nh * npairs;
  if (ncl > ctx->max_pairs) ncl = ctx->max_pairs;
  cfg.gridDim = dim3(2 * ncl);
  int Mi = (int)M, nh = c.nh, H = c.hidden, q_early = ctx->apply_q_early;
  cudaError_t e = cudaLaunchKernelEx(&cfg, bf16_apply_wide_pair_kernel, mapW, mapQ, O, Mi, ld, nh, H, npairs, q_early);
  if (e != cudaSuccess) return set_error(ctx, TTT_ERR_CUDA, "bf16_apply_wide_pair_kernel launch", e);
  TTT_LAUNCH_CHECK(ctx, "bf16_apply_wide_pair_kernel");
  return TTT_OK;
}

}  // namespace ttt
