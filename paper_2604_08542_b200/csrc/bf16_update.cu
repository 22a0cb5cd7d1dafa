// bf16_update.cu — fused tensor-core gradient kernel of the TTT update (steps 1-5 of the hot path,
// DESIGN.md "Kernels"; Eq. 8 with Eq. 9 and Eq. 12).
//
// Formulation ("hidden on lanes"): one CTA owns 128 hidden units of one head and a range of tokens.
// Everything is computed TRANSPOSED so that each MMA has M = 128 hidden units on the TMEM lanes:
//   forward   x^T  = (W1/2)^T K^T,  b^T = W3^T K^T,  g0^T = W2 V^T   [128 x T]  (contract over hd)
//             g = -eta g0 = dHd (dot-product loss: dL/df = -eta v, Eq. 9)
//   epilogue  th = tanh(x);  S = x + x th = SiLU(a);  t = (1 + th) + S (1 - th) = 2 SiLU'(a)
//             dA2 = g b t (= 2 dA);  dB = g S;  Hd' = -eta S b                 (fp32 -> fp16)
//   gradient  2 G1^T += dA2^T K,  G3^T += dB^T K,  G2 += Hd'^T V     [128 x hd] (contract over tokens)
// The A operand of every MMA lives in TMEM (weights: loaded once, W1 pre-halved (exact) so the
// accumulator is the tanh argument; dA2/dB/Hd: written by the epilogue over their own fp32 sources),
// the B operand is the K or V token tile in shared memory with the 128-byte swizzle; the SAME tile
// serves the forward MMA as a K-major operand and the gradient MMA as an MN-major operand, so the
// shared-memory operand traffic is 64 B/clk at tensor peak. Gradient accumulators stay in TMEM for
// the CTA's whole token range; one fp32 partial per CTA goes to L2 and is summed in a fixed order
// by the commit (deterministic, no float atomics). The factor 2 of G1 is removed at the flush.
//
// Warp roles (640 threads): warp 0 = TMA producer; warp 1 = forward-MMA issuer; warp 2 = learning-
// rate loader (-eta of a tile into the stage's shared-memory slot, prefetched ahead of the ring; scaling
// V in shared memory instead costs a serial read-modify-write + proxy fence per tile); warp 3 = gradient-MMA
// issuer (two issuers: an mbarrier wait costs ~90 clk even when already complete, and MMA issue
// blocks at the tensor pipe's pace, so one thread cannot keep the pipe fed); warps 4-19 = two
// epilogue groups of 8 warps that alternate token tiles (2 warps per TMEM lane quarter, one
// 16-token K step each; packed fp32x2 math, tanh.approx sigmoid).
// Pipeline (TMEM is the scarce resource: weights 96 + gradient accumulators 192 columns leave 224):
// the x | b forward accumulators are double-buffered, g is single-buffered and released first, as
// soon as an epilogue group has pulled it into registers; the fp16 gradient operands have their own
// (single) columns, so nothing aliases; forward and gradient MMAs are issued by different warps —
// the MMAs of tiles i+1, i+2 overlap the epilogue math of tile i.
// Measured budget per 32-token tile and SM (B200 microbenchmarks): tensor pipe 384 clk
// when the twelve N=32 and six N=64 MMAs are issued back to back (nominal rate), epilogue math
// ~390 clk (MUFU 16/clk: 256; FP32 pipe 128 lanes/clk: 10 ops per element; F2FP packs). The kernel
// runs at ~786 clk per tile: the forward-issuing thread's own instruction stream (~100 dependent
// scalar instructions per tile around the twelve MMAs) plus the single-buffered g hand-off are the
// critical path — variants that split or re-home that stream measured slower.
#include <stdio.h>

#include "tc_common.cuh"
#include "ttt_internal.h"

namespace ttt {

namespace upd {
constexpr int HS = 128;        // hidden units per CTA (MMA M)
constexpr int T = 32;          // tokens per tile (forward MMA N, gradient MMA K)
constexpr int STAGES = 10;     // K/V shared-memory ring (ring latency = TMA + F -> E -> G hand-offs)
constexpr int EPI_WARPS = 16;
constexpr int CVT_WARPS = 2;   // stage finishers: warps 0 and 2
// 20 warps: 5 per scheduler keep 96 registers per thread (a 21st warp caps everybody at 80 and the
// epilogue spills)
constexpr int THREADS = (4 + EPI_WARPS) * 32;
constexpr int TILE_BYTES = T * 128;  // one [T x 64] bf16 tile
constexpr int STAGE_BYTES = 2 * TILE_BYTES;

// TMEM column plan for hd = 64 (512 columns x 128 lanes x 32 bit)
constexpr uint32_t C_W1 = 0, C_W3 = 32, C_W2 = 64;        // fp16 weights as A operands, 32 cols each
constexpr uint32_t C_G1 = 96, C_G3 = 160, C_G2 = 224;     // fp32 gradient accumulators, 64 cols each
constexpr uint32_t C_XB = 288, XB_STRIDE = 64;            // two forward buffers x | b (fp32, 32 cols each)
constexpr uint32_t C_GG = 416;                            // forward accumulator g (fp32, 32 cols), single
constexpr uint32_t C_H = 448;                             // fp16 operands dA2 | dB | Hd, 16 cols each, single
}  // namespace upd

template <bool LOSS>
__global__ void __launch_bounds__(upd::THREADS, 1)
bf16_update_kernel(const __grid_constant__ CUtensorMap mapK, const __grid_constant__ CUtensorMap mapV,
                   const ttt_wop_t* __restrict__ Wb, const float* __restrict__ lr,
                   float* __restrict__ P, float* __restrict__ loss_part, int M, int nh, int H,
                   int tiles_total, int tiles_per_split, float* __restrict__ Wm,
                   ttt_wop_t* __restrict__ Wbw, unsigned* __restrict__ sync_ctr,
                   unsigned sync_target, const float* __restrict__ renorm_n0,
                   float* __restrict__ renorm_colsq) {
  using namespace upd;
  constexpr int HD = 64;
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  // 1024-B aligned base, computed on the 32-bit shared-space address (a uniform value)
  const uint32_t sbase = (smem_u32(smem_raw) + 1023u) & ~1023u;
  uint8_t* smem = smem_raw + (sbase - smem_u32(smem_raw));
  __shared__ uint64_t tma_full[STAGES], full[STAGES], empty[STAGES], fwd_full[2], xb_free[2], g_free,
      epi_done[2], opnd_free[2], w_ready, grad_done;
  __shared__ uint32_t tmem_base_s;
  __shared__ float loss_red[EPI_WARPS];
  __shared__ float lrmax_s[THREADS / 32];
  static_assert(THREADS % 16 == 0, "the fused commit gives 16 lanes one weight row");
  __shared__ __align__(16) float ne_s[STAGES][T];   // -eta of the stage's tokens, scaled (0 beyond M)

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int split = blockIdx.x, slice = blockIdx.y, h = blockIdx.z;
  const int nslices = gridDim.y;
  const int tile_lo = split * tiles_per_split;
  const int ntiles = min(tiles_per_split, tiles_total - tile_lo);

  // Prologue, spread over three threads so that nothing queues behind anything else: the first
  // TMA round trip (descriptor fetch + HBM, ~2 us = 3.5 K clk) is the critical path of the start-up,
  // so thread 0 initialises only the ring's `full` barriers and requests the first ring of K/V tiles;
  // warp 1 initialises the other barriers; warp 3 allocates TMEM (trace, r01e: requests left at
  // 2.3-3.6 K clk when all of this was serial in thread 0, first forward MMA at 7-9 K clk).
  if (tid == 0) {
    tma_prefetch_desc(&mapK);
    tma_prefetch_desc(&mapV);
#pragma unroll
    for (int s = 0; s < STAGES; ++s) mbar_init(&tma_full[s], 1);
    fence_mbar_init();
    const int npre = min(ntiles, STAGES);
    for (int i = 0; i < npre; ++i) {
      mbar_arrive_expect_tx(&tma_full[i], STAGE_BYTES);
      uint8_t* dst = smem + i * STAGE_BYTES;
      tma_load_2d(dst, &mapK, &tma_full[i], h * HD, (tile_lo + i) * T);
      tma_load_2d(dst + TILE_BYTES, &mapV, &tma_full[i], h * HD, (tile_lo + i) * T);
    }
  } else if (tid == 32) {
#pragma unroll
    for (int s = 0; s < STAGES; ++s) { mbar_init(&empty[s], 1); mbar_init(&full[s], CVT_WARPS); }
    mbar_init(&fwd_full[0], 1);
    mbar_init(&fwd_full[1], 1);
    mbar_init(&g_free, EPI_WARPS / 2);
    mbar_init(&opnd_free[0], 1);
    mbar_init(&opnd_free[1], 1);
    for (int b = 0; b < 2; ++b) { mbar_init(&epi_done[b], EPI_WARPS / 2); mbar_init(&xb_free[b], EPI_WARPS / 2); }
    mbar_init(&w_ready, EPI_WARPS);
    mbar_init(&grad_done, 1);
    fence_mbar_init();
  }
  __syncwarp();
  // epilogue warps request their share of the fp16 weights now (row j of W1^T, W2, W3^T; 16-byte
  // chunks 2 tc, 2 tc + 1), so the L2 latency overlaps the TMEM allocation
  uint4 wpre[3][2];
  if (warp >= 4) {
    const int tc_ = (warp - 4) >> 2, j_ = (warp & 3) * 32 + lane;
    const size_t me_ = (size_t)nh * H * HD;
    const size_t row_ = ((size_t)h * H + (size_t)slice * HS + j_) * HD;
#pragma unroll
    for (int mat = 0; mat < 3; ++mat) {
      const uint4* src = reinterpret_cast<const uint4*>(Wb + mat * me_ + row_) + 2 * tc_;
      wpre[mat][0] = __ldg(src);
      wpre[mat][1] = __ldg(src + 1);
    }
  }
  // ... and the learning-rate loader its first batch (cold HBM latency off the first tile's path)
  constexpr int LRPF = 8;
  float lr_pre[LRPF];
  if (warp == 2) {
#pragma unroll
    for (int u = 0; u < LRPF; ++u) {
      const int t = (tile_lo + u) * T + lane;
      lr_pre[u] = (u < ntiles && t < M) ? __ldg(lr + (size_t)h * M + t) : 0.f;   // negated after the barrier
    }
  }
  // max |eta| over the CTA's token range (all threads; the loads overlap the first TMA round trip)
  {
    const float* lrh = lr + (size_t)h * M;
    const int t_hi = min(M, (tile_lo + ntiles) * T);
    float mx = 0.f;
#pragma unroll 4
    for (int t = tile_lo * T + tid; t < t_hi; t += THREADS) mx = fmaxf(mx, fabsf(__ldg(lrh + t)));
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    if (lane == 0) lrmax_s[warp] = mx;
  }
  if (warp == 3) { tmem_alloc(&tmem_base_s, 512); tmem_relinquish(); }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tb = tmem_base_s;
  if (tb != 0) __trap();      // all 512 columns belong to this CTA: the issuers use absolute columns
  float eta_sc, eta_isc;      // the gradient operands carry eta * eta_sc; undone at the flush
  {
    float mx = 0.f;
#pragma unroll
    for (int w = 0; w < THREADS / 32; ++w) mx = fmaxf(mx, lrmax_s[w]);
    eta_scale(mx, eta_sc, eta_isc);
  }

  if (warp == 0) {
    // ===================== stage finisher 1: fp16 conversion (second half of a stage) =====================
    // (tiles 0 .. STAGES-1 were requested by thread 0 in the prologue; the gradient issuer refills the ring)
    for (int i = 0; i < ntiles; ++i) {
      const int s = i % STAGES;
      mbar_wait(&tma_full[s], (i / STAGES) & 1);
      tile_bf16_to_f16<STAGE_BYTES / 512 / CVT_WARPS>(smem + s * STAGE_BYTES + STAGE_BYTES / CVT_WARPS, lane);
      fence_proxy_async_smem();
      __syncwarp();
      if (lane == 0) mbar_arrive(&full[s]);
    }
  } else if (warp == 1) {
    // ===================== forward-MMA issuer =====================
    // One elected thread runs the whole loop; it is bound by its own serial instruction stream, so
    // everything it needs per tile is a constant or an increment: the CTA owns all 512 TMEM columns
    // (base 0, checked above), stage descriptors advance by a fixed step, phases are flipped bits.
    if (elect_one()) {
      constexpr uint32_t idesc_f = umma_idesc(HS, T, 0, 0, TTT_FMT_F16, TTT_FMT_F16);   // A = weights, B = token tile (fp16), K-major
      constexpr uint32_t V_OFF = TILE_BYTES >> 4, ST_OFF = STAGE_BYTES >> 4;   // descriptor steps (16-B units)
      const uint64_t d0 = umma_smem_desc_sw128(sbase, 16, 1024);
      mbar_wait(&w_ready, 0);
      tc_fence_after();
      int s = 0;
      uint32_t ph_full = 0;
      uint64_t dk = d0;
      for (int i = 0; i < ntiles; ++i) {
        const int b = i & 1, n = i >> 1;
        // the waits of a tile are probed together (a probe costs ~90 clk even when the phase is
        // already complete), then re-waited only if a probe failed
        const uint32_t ok0 = mbar_try_wait(&full[s], ph_full);
        const uint32_t ok1 = n > 0 ? mbar_try_wait(&xb_free[b], (n - 1) & 1) : 1u;
        const uint32_t ok2 = i > 0 ? mbar_try_wait(&g_free, (i - 1) & 1) : 1u;
        if (!ok0) mbar_wait(&full[s], ph_full);
        if (!ok1) mbar_wait(&xb_free[b], (n - 1) & 1);
        tc_fence_after();
        const uint32_t acc = C_XB + b * XB_STRIDE;
#pragma unroll
        for (int k = 0; k < HD / 16; ++k) umma_ts(acc, C_W1 + 8 * k, dk + 2 * k, idesc_f, k > 0);
#pragma unroll
        for (int k = 0; k < HD / 16; ++k) umma_ts(acc + 32, C_W3 + 8 * k, dk + 2 * k, idesc_f, k > 0);
        if (!ok2) { mbar_wait(&g_free, (i - 1) & 1); tc_fence_after(); }   // g of tile i-1 is in registers
#pragma unroll
        for (int k = 0; k < HD / 16; ++k) umma_ts(C_GG, C_W2 + 8 * k, dk + V_OFF + 2 * k, idesc_f, k > 0);
        tc_commit(&fwd_full[b]);   // one barrier per epilogue group: a parity wait only tells the
                                   // current phase from the previous one
        if (++s == STAGES) { s = 0; ph_full ^= 1; dk = d0; } else { dk += ST_OFF; }
      }
    }
  } else if (warp == 3) {
    // ===================== gradient-MMA issuer =====================
    if (elect_one()) {
      constexpr uint32_t idesc_g = umma_idesc(HS, HD, 0, 1, TTT_FMT_F16, TTT_FMT_F16);   // A = fp16 operands, B = token tile (fp16), MN-major
      constexpr uint32_t V_OFF = TILE_BYTES >> 4, ST_OFF = STAGE_BYTES >> 4;
      const uint64_t d0 = umma_smem_desc_sw128(sbase, TILE_BYTES, 1024);
      int s = 0;
      uint64_t dk = d0;
      for (int i = 0; i < ntiles; ++i) {
        const int b = i & 1, n = i >> 1;
        mbar_wait(&epi_done[b], n & 1);
        tc_fence_after();
        const uint32_t acc_flag = i > 0;
#pragma unroll
        for (int k = 0; k < T / 16; ++k)                     // +2048 B per 16-token K step
          umma_ts(C_G1, C_H + 8 * k, dk + 128 * k, idesc_g, acc_flag | k);
#pragma unroll
        for (int k = 0; k < T / 16; ++k)
          umma_ts(C_G3, C_H + 16 + 8 * k, dk + 128 * k, idesc_g, acc_flag | k);
#pragma unroll
        for (int k = 0; k < T / 16; ++k)
          umma_ts(C_G2, C_H + 32 + 8 * k, dk + V_OFF + 128 * k, idesc_g, acc_flag | k);
        tc_commit(&empty[s]);          // the tile's forward MMAs completed long ago (epilogue read them)
        tc_commit(&opnd_free[b]);     // one barrier per tile parity (see the epilogue's wait)
        // TMA producer duty (this thread has the slack; warp 0 is a stage finisher): the stage of tile
        // i - 1, whose gradient MMAs were issued an iteration ago and are normally complete by now, is
        // refilled with tile i - 1 + STAGES
        if (i >= 1 && i - 1 + STAGES < ntiles) {
          const int j = i - 1 + STAGES, sj = (i - 1) % STAGES;
          mbar_wait(&empty[sj], ((i - 1) / STAGES) & 1);
          mbar_arrive_expect_tx(&tma_full[sj], STAGE_BYTES);
          uint8_t* dst = smem + sj * STAGE_BYTES;
          tma_load_2d(dst, &mapK, &tma_full[sj], h * HD, (tile_lo + j) * T);
          tma_load_2d(dst + TILE_BYTES, &mapV, &tma_full[sj], h * HD, (tile_lo + j) * T);
        }
        if (++s == STAGES) { s = 0; dk = d0; } else { dk += ST_OFF; }
      }
      tc_commit(&grad_done);
    }
  } else if (warp == 2) {
    // ===================== stage finisher 0: fp16 conversion + learning rates =====================
    // When the TMA has landed a stage, the two finisher warps (this one: the K tile, warp 0: the V tile)
    // convert it from bf16 to fp16 in place (all MMA operands are fp16, ttt_internal.h; one warp alone
    // needs 550-750 clk per stage next to the epilogue warps of its scheduler and becomes the kernel's
    // critical path), and this one also puts
    // -eta of the tile's 32 tokens (one 128-B line of lr, scaled by the CTA's power of two) into the
    // stage's slot; the stage is `full` when all of them have arrived. The global loads of lr run LRPF
    // tiles ahead of the ring (register double buffer).
    const float* lrh = lr + (size_t)h * M;
    auto ld_batch = [&](int i0, float (&v)[LRPF]) {
#pragma unroll
      for (int u = 0; u < LRPF; ++u) {
        const int t = (tile_lo + i0 + u) * T + lane;
        v[u] = (i0 + u < ntiles && t < M) ? -eta_sc * __ldg(lrh + t) : 0.f;
      }
    };
    float cur[LRPF], nxt[LRPF];
#pragma unroll
    for (int u = 0; u < LRPF; ++u) cur[u] = -eta_sc * lr_pre[u];   // requested before the allocation barrier
    for (int i0 = 0; i0 < ntiles; i0 += LRPF) {
      ld_batch(i0 + LRPF, nxt);
#pragma unroll
      for (int u = 0; u < LRPF; ++u) {
        const int i = i0 + u;
        if (i < ntiles) {
          const int s = i % STAGES, it = i / STAGES;
          mbar_wait(&tma_full[s], it & 1);       // (the TMA was issued after the stage's `empty`)
          tile_bf16_to_f16<STAGE_BYTES / 512 / CVT_WARPS>(smem + s * STAGE_BYTES, lane);
          ne_s[s][lane] = cur[u];
          fence_proxy_async_smem();
          __syncwarp();
          if (lane == 0) mbar_arrive(&full[s]);

        }
      }
#pragma unroll
      for (int u = 0; u < LRPF; ++u) cur[u] = nxt[u];
    }
  } else {
    // ===================== epilogue warps =====================
    const int ew = warp - 4, q = warp & 3;
    const int grp = ew >> 3, kh = (ew >> 2) & 1;           // tile parity this warp serves, K step (16 tokens)
    const int tc = ew >> 2;                                // 16-column group for the weight load / flush
    const int j = q * 32 + lane;                           // hidden unit within the slice = TMEM lane
    const uint32_t lane_base = static_cast<uint32_t>(q * 32) << 16;
    const size_t me = (size_t)nh * H * HD;
    const size_t row = ((size_t)h * H + (size_t)slice * HS + j) * HD;
    {
      // weights -> TMEM as A operands: row j of W1^T / 2, W3^T, W2 (64 fp16 = 32 words each); warp
      // group tc loads 16-byte chunks 2 tc, 2 tc + 1 of each row (8 words = columns 8 tc .. 8 tc + 7)
      const uint32_t cols[3] = {C_W1, C_W2, C_W3};
      uint4 (&x)[3][2] = wpre;           // requested before the TMEM allocation barrier
#pragma unroll
      for (int mat = 0; mat < 3; ++mat) {
        uint32_t r[8] = {x[mat][0].x, x[mat][0].y, x[mat][0].z, x[mat][0].w,
                         x[mat][1].x, x[mat][1].y, x[mat][1].z, x[mat][1].w};
        if (mat == 0) {
#pragma unroll
          for (int e = 0; e < 8; ++e) {    // W1 / 2: the accumulator becomes the tanh argument a / 2
            const float2 f = __half22float2(*reinterpret_cast<const __half2*>(&r[e]));
            r[e] = pack_f16x2(0.5f * f.x, 0.5f * f.y);
          }
        }
        tmem_st_x8(tb + lane_base + cols[mat] + 8 * tc, r);
      }
      tc_wait_st();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&w_ready);
    }
    uint64_t loss2 = 0ull;
    const uint64_t ONE2 = pack2(1.0f, 1.0f), NONE2 = pack2(-1.0f, -1.0f);
    const uint32_t xbuf = tb + lane_base + C_XB + grp * XB_STRIDE + 16 * kh;
    const uint32_t gbuf = tb + lane_base + C_GG + 16 * kh;
    const uint32_t hbuf = tb + lane_base + C_H + 8 * kh;
    for (int i = grp; i < ntiles; i += 2) {
      const int n = i >> 1;
      mbar_wait(&fwd_full[grp], n & 1);
      mbar_wait(&full[i % STAGES], (i / STAGES) & 1);      // direct acquire of the loader's -eta slot
      tc_fence_after();
      const uint2* nes = reinterpret_cast<const uint2*>(&ne_s[i % STAGES][16 * kh]);
      uint32_t rx[16], rb[16], rg[16];
      tmem_ld_x16(gbuf, rg);                               // g is single-buffered: release it first
      tc_wait_ld();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&g_free);
      tmem_ld_x16(xbuf, rx);
      tmem_ld_x16(xbuf + 32, rb);
      tc_wait_ld();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&xb_free[grp]);           // forward MMAs of tile i+2 may overwrite x | b
      uint32_t pa[8], pb[8], ph[8];
#pragma unroll
      for (int c = 0; c < 16; c += 2) {
        const uint64_t x = pack2u(rx[c], rx[c + 1]);
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
      // the operand buffer was last read by the gradient MMAs of tile i - 1
      // (an epilogue group sees every OTHER tile: on one barrier shared by both tile parities its
      // parity wait could not tell "tile i - 1 done" from "tile i - 3 done" when the gradient issuer
      // lags by two tiles, and a fast warp would overwrite operands not yet read; with one barrier per
      // tile parity the phase it waits for is always the barrier's current or latest completed one)
      if (i > 0) { mbar_wait(&opnd_free[grp ^ 1], ((i - 1) >> 1) & 1); tc_fence_after(); }
      tmem_st_x8(hbuf, pa);
      tmem_st_x8(hbuf + 16, pb);
      tmem_st_x8(hbuf + 32, ph);
      tc_wait_st();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&epi_done[grp]);
    }
    // a dependent kernel (PDL) may be scheduled from here on; it still waits for this grid to finish
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    // ---- flush the gradient accumulators: one fp32 partial slice per CTA ----
    mbar_wait(&grad_done, 0);
    tc_fence_after();
    float* Pset = P + (size_t)split * 3 * me;
    const uint32_t gcol[3] = {C_G1, C_G2, C_G3};
    // TMEM gives a thread 16 columns of ONE row: written to global memory directly, a warp store would
    // touch 32 lines for 512 bytes (measured: 6.3 K clk for the flush). The idle K/V ring stages each
    // matrix as [128][68] fp32 (two buffers, alternating), then the slice's 32 KB leave as full lines.
    constexpr int SLD = HD + 4;
    float* stg = reinterpret_cast<float*>(smem);
    const int et = ew * 32 + lane;                         // 0 .. 511
    const size_t slice_base = ((size_t)h * H + (size_t)slice * HS) * HD;
#pragma unroll
    for (int mat = 0; mat < 3; ++mat) {                    // this warp: columns 16 tc .. 16 tc + 15
      uint32_t r[16];
      if (ntiles > 0) {
        tmem_ld_x16(tb + lane_base + gcol[mat] + 16 * tc, r);
        tc_wait_ld();
      } else {
#pragma unroll
        for (int u = 0; u < 16; ++u) r[u] = 0u;
      }
      const float sc = (mat == 0 ? 0.5f : 1.0f) * eta_isc; // G1 was accumulated from 2 dA; eta scale undone
      float* sb = stg + (mat & 1) * HS * SLD;
      float4* d = reinterpret_cast<float4*>(sb + j * SLD + 16 * tc);
#pragma unroll
      for (int v = 0; v < 4; ++v)
        d[v] = make_float4(sc * __uint_as_float(r[4 * v]), sc * __uint_as_float(r[4 * v + 1]),
                           sc * __uint_as_float(r[4 * v + 2]), sc * __uint_as_float(r[4 * v + 3]));
      asm volatile("bar.sync 9, 512;" ::: "memory");
      float4* dst = reinterpret_cast<float4*>(Pset + mat * me + slice_base);
#pragma unroll
      for (int k = 0; k < HS * HD / 4 / 512; ++k) {
        const int e = et + 512 * k;                        // float4 index: row e / 16, columns 4 (e % 16)
        dst[e] = *reinterpret_cast<const float4*>(sb + (e >> 4) * SLD + 4 * (e & 15));
      }
    }
    if (LOSS) {
      float l0, l1;
      unpack2(loss2, l0, l1);
      float loss = l0 + l1;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) loss += __shfl_xor_sync(0xffffffffu, loss, o);
      if (lane == 0) loss_red[ew] = loss;
      asm volatile("bar.sync 9, 512;" ::: "memory");
      if (ew == 0 && lane == 0) {
        float t = 0.f;
        for (int w = 0; w < EPI_WARPS; ++w) t += loss_red[w];
        loss_part[((size_t)split * nslices + slice) * nh + h] = t * eta_isc;
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 3) tmem_dealloc(tb, 512);
  if (Wm != nullptr) {
    // ---- fused commit (Eq. 8): W <- W - sum_s P[s], summed in split order [+ re-normalisation] ----
    // The `gridDim.x` CTAs that share this (head, slice) meet at a counter in global memory (the
    // launch is cooperative: all CTAs are resident), then each commits its share of the slice's
    // 3 x 128 rows: fp32 master + fp16 operand copy. Deterministic: fixed summation order.
    const int nsplit = gridDim.x;
    if (tid == 0) {
      __threadfence();
      atomicAdd(&sync_ctr[h * nslices + slice], 1u);
      unsigned v;
      long long t0 = clock64();
      do {
        asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(sync_ctr + h * nslices + slice) : "memory");
        if (clock64() - t0 > TTT_MBAR_TIMEOUT_CYCLES) __trap();
      } while ((int)(v - sync_target) < 0);
    }
    __syncthreads();
    const size_t me = (size_t)nh * H * HD, set = 3 * me;
    const size_t row0 = ((size_t)h * H + (size_t)slice * HS) * HD;
    constexpr int N4 = 3 * HS * HD / 4;                     // float4 per slice
    constexpr int RQ = HD / 4;                              // float4 per row (16 lanes own one row)
    const int chunk = ((N4 + nsplit - 1) / nsplit + RQ - 1) / RQ * RQ;   // whole rows per CTA
    const int e_lo = min(N4, split * chunk), e_hi = min(N4, e_lo + chunk);
    float4 colacc = make_float4(0.f, 0.f, 0.f, 0.f);        // renorm: W2 column sums of squares
    // The loop is bound by L2 round trips (~700 clk each under load), so a pass covers CE elements
    // per thread and requests CU partial sets of each at once: nsplit = 9 (cfg2: 688 float4 per CTA)
    // takes 2 round trips, nsplit = 4 (cfg3/cfg4: 1536) 2 passes of one (trace, r01e: 5.7 K clk for
    // the one-element, four-sets-at-a-time loop at cfg2). The sum keeps the split order.
    constexpr int CE = 2, CU = 5;
    for (int base = e_lo; base < e_hi; base += CE * THREADS) {   // THREADS % 16 == 0: a lane keeps its columns
      bool ok[CE];
      int mat[CE], r4[CE];
      size_t off[CE];
      float4 w[CE], g[CE];
#pragma unroll
      for (int k = 0; k < CE; ++k) {
        const int e = base + k * THREADS + tid;
        ok[k] = e < e_hi;
        mat[k] = ok[k] ? e / (HS * HD / 4) : 0;
        r4[k] = ok[k] ? e % (HS * HD / 4) : 0;
        off[k] = mat[k] * me + row0 + (size_t)r4[k] * 4;
        w[k] = make_float4(0.f, 0.f, 0.f, 0.f);
        g[k] = make_float4(0.f, 0.f, 0.f, 0.f);
        if (ok[k]) w[k] = *reinterpret_cast<const float4*>(Wm + off[k]);
      }
      for (int sp0 = 0; sp0 < nsplit; sp0 += CU) {
        float4 p[CE][CU];
#pragma unroll
        for (int k = 0; k < CE; ++k)
#pragma unroll
          for (int u = 0; u < CU; ++u)
            if (ok[k] && sp0 + u < nsplit)
              p[k][u] = __ldcg(reinterpret_cast<const float4*>(P + (size_t)(sp0 + u) * set + off[k]));
#pragma unroll
        for (int k = 0; k < CE; ++k)
#pragma unroll
          for (int u = 0; u < CU; ++u)
            if (ok[k] && sp0 + u < nsplit) {
              if (sp0 + u == 0) g[k] = p[k][u];
              else { g[k].x += p[k][u].x; g[k].y += p[k][u].y; g[k].z += p[k][u].z; g[k].w += p[k][u].w; }
            }
      }
#pragma unroll
      for (int k = 0; k < CE; ++k) {
        if (ok[k]) { w[k].x -= g[k].x; w[k].y -= g[k].y; w[k].z -= g[k].z; w[k].w -= g[k].w; }
        if (renorm_n0 != nullptr) {
          // row sums of squares: every lane of the warp takes part in the shuffles (lanes beyond e_hi
          // carry w = 0) — a warp may straddle a matrix boundary or the end of the CTA's range, while
          // the 16 lanes of one row always share `ok` and `mat`
          float sq = w[k].x * w[k].x + w[k].y * w[k].y + w[k].z * w[k].z + w[k].w * w[k].w;
#pragma unroll
          for (int o = RQ / 2; o > 0; o >>= 1) sq += __shfl_xor_sync(0xffffffffu, sq, o);
          if (ok[k] && mat[k] != 1) {   // W1^T / W3^T: a row is a unit's fan-in vector -> back to its initial norm
            const int j = slice * HS + r4[k] / RQ;
            const float* n0m = renorm_n0 + (mat[k] == 0 ? (size_t)h * H : (size_t)nh * H + (size_t)nh * HD + (size_t)h * H);
            const float f = n0m[j] / (sqrtf(sq) + 1e-5f);
            w[k].x *= f; w[k].y *= f; w[k].z *= f; w[k].w *= f;
          } else if (ok[k]) {   // W2: fan-in = column; finished by renorm_w2_kernel from per-CTA partials
            colacc.x = fmaf(w[k].x, w[k].x, colacc.x); colacc.y = fmaf(w[k].y, w[k].y, colacc.y);
            colacc.z = fmaf(w[k].z, w[k].z, colacc.z); colacc.w = fmaf(w[k].w, w[k].w, colacc.w);
          }
        }
        if (ok[k]) {
          *reinterpret_cast<float4*>(Wm + off[k]) = w[k];
          *reinterpret_cast<uint2*>(Wbw + off[k]) = make_uint2(ttt_pack_wop2(w[k].x, w[k].y), ttt_pack_wop2(w[k].z, w[k].w));
        }
      }
    }
    if (renorm_n0 != nullptr) {
      float4* cs = reinterpret_cast<float4*>(smem);         // the K/V ring is idle by now
      cs[tid] = colacc;
      __syncthreads();
      if (tid < RQ) {
        float4 t = make_float4(0.f, 0.f, 0.f, 0.f);
        for (int r = 0; r < THREADS / RQ; ++r) {            // fixed order
          const float4 v = cs[r * RQ + tid];
          t.x += v.x; t.y += v.y; t.z += v.z; t.w += v.w;
        }
        const int nblk = nslices * nsplit;
        *reinterpret_cast<float4*>(renorm_colsq + ((size_t)h * nblk + slice * nsplit + split) * HD + 4 * tid) = t;
      }
    }
  }
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
  if (ctx->large) return 0;            // the gradient GEMMs write the dense gradient
  if (ctx->cfg.hd == 128) return bf16_wide_partials_needed(ctx, M);
  int a, b, s;
  update_split(ctx, M, &a, &b, &s);
  return s;
}

static int narrow_tensor_path(const ttt_config* cfg) {
  return cfg->hd == 64 && (cfg->hidden == 128 || cfg->hidden == 256) && !cfg->linear_fast_weight;
}
int bf16_apply_tensor_path(const ttt_config* cfg) {
  return narrow_tensor_path(cfg) || bf16_apply_wide_supported(cfg) || bf16_large_supported(cfg);
}
int bf16_update_tensor_path(const ttt_config* cfg) {
  return narrow_tensor_path(cfg) || bf16_update_wide_supported(cfg) || bf16_large_supported(cfg);
}

// Shapes the bf16 <-> fp32 conversion in front of the fp32 CUDA-core kernels can take at all; whether a
// bf16 shape is ACCEPTED is decided in ttt_create: a tcgen05 kernel exists (bf16_*_tensor_path), or the
// caller opted in with cfg.cuda_core_fallback (same semantics, fp32 arithmetic).
int bf16_supported(const ttt_config* cfg, char* why, size_t why_len) {
  if (cfg->linear_fast_weight) { snprintf(why, why_len, "bf16 path: linear test mode is f32-only"); return 0; }
  if (cfg->hd % 8 != 0) { snprintf(why, why_len, "bf16 path: hd must be a multiple of 8 (got %d)", cfg->hd); return 0; }
  return 1;
}

int bf16_accumulate(ttt_ctx* ctx, const __nv_bfloat16* K, const __nv_bfloat16* V, const float* lr,
                    int64_t M, int64_t ld, bool want_loss, bool fuse_commit, int* used, int* loss_rows,
                    cudaStream_t s) {
  const ttt_config& c = ctx->cfg;
  int tiles, tps, splits;
  update_split(ctx, M, &tiles, &tps, &splits);
  if (c.hd == 128)                       // hd = 128: weights in shared memory, no fused commit
    return bf16_accumulate_wide(ctx, K, V, lr, M, ld, want_loss, used, loss_rows, s);
  CUtensorMap mapK, mapV;
  int rc = make_token_map(ctx, &mapK, K, M, (int64_t)c.nh * c.hd, ld, upd::T);
  if (rc != TTT_OK) return rc;
  rc = make_token_map(ctx, &mapV, V, M, (int64_t)c.nh * c.hd, ld, upd::T);
  if (rc != TTT_OK) return rc;
  const size_t smem = (size_t)upd::STAGES * upd::STAGE_BYTES + 1024;
  if (!(ctx->attr_done & ATTR_UPD)) {
    TTT_CUDA_TRY(ctx, cudaFuncSetAttribute(bf16_update_kernel<false>,
                                           cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem),
                 "bf16_update_kernel smem attr");
    TTT_CUDA_TRY(ctx, cudaFuncSetAttribute(bf16_update_kernel<true>,
                                           cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem),
                 "bf16_update_kernel smem attr");
    int per_sm = 0;            // CTAs the device can really hold at once (MPS / green contexts shrink it)
    TTT_CUDA_TRY(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, bf16_update_kernel<false>,
                                                                    upd::THREADS, smem),
                 "bf16_update_kernel occupancy");
    ctx->upd_coop_ctas = per_sm * ctx->sm_count;
    ctx->attr_done |= ATTR_UPD;
  }
  const int nslices = c.hidden / upd::HS;
  float* P = ctx->partials + (size_t)ctx->n_partials * 3 * ctx->mat_elems;
  dim3 grid(splits, nslices, c.nh);
  // fused commit: the CTAs of a (head, slice) group wait on one another, so they must all be
  // resident -> cooperative launch, only when the device can hold the whole grid; if that launch is
  // refused all the same, the plain launch + commit kernel path below is taken (same results)
  fuse_commit = fuse_commit && (int)(grid.x * grid.y * grid.z) <= ctx->upd_coop_ctas;
  const ttt_wop_t* Wb = ctx->Wb;
  float* loss_part = ctx->loss_part;
  int Mi = (int)M, nh = c.nh, H = c.hidden;
  unsigned* ctr = ctx->sync_ctr;
  float* rcs = ctx->colsq;
  const void* fn = want_loss ? (const void*)bf16_update_kernel<true> : (const void*)bf16_update_kernel<false>;
  for (;;) {
    float* Wm = fuse_commit ? ctx->Wm : nullptr;
    ttt_wop_t* Wbw = fuse_commit ? ctx->Wb : nullptr;
    unsigned target = ctx->sync_target + (fuse_commit ? (unsigned)splits : 0u);
    const float* rn0 = (fuse_commit && c.renorm) ? ctx->n0 : nullptr;
    void* args[] = {&mapK, &mapV, &Wb, &lr, &P, &loss_part, &Mi, &nh, &H, &tiles, &tps, &Wm, &Wbw, &ctr,
                    &target, &rn0, &rcs};
    cudaError_t e = fuse_commit ? cudaLaunchCooperativeKernel(fn, grid, dim3(upd::THREADS), args, smem, s)
                                : cudaLaunchKernel(fn, grid, dim3(upd::THREADS), args, smem, s);
    if (e == cudaSuccess) {
      ctx->sync_target = target;         // only a launch that happened moves the counters' target
      break;
    }
    if (!fuse_commit) return set_error(ctx, TTT_ERR_CUDA, "bf16_update_kernel launch", e);
    cudaGetLastError();                  // cooperative launch refused: clear it, take the plain path
    fuse_commit = false;
  }
  TTT_LAUNCH_CHECK(ctx, "bf16_update_kernel");
  *used = fuse_commit ? 0 : splits;
  *loss_rows = splits * nslices;
  if (fuse_commit && c.renorm) {       // W2's column fan-in norms span the head's slices: finish them
    rc = launch_renorm_w2(ctx, nslices * splits, s);
    if (rc != TTT_OK) return rc;
  }
  return fuse_commit ? 1 : TTT_OK;     // 1 = gradient already committed by the kernel
}

}  // namespace ttt
