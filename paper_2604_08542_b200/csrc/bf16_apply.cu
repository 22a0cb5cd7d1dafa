// bf16_apply.cu — fused tensor-core apply kernel (steps 9-11 of the hot path):
//   O = ( SiLU(Q W1) o (Q W3) ) W2        Eq. 4 with Eq. 12, updated weights.
//
// Formulation ("tokens on lanes"): a CTA owns one head and a strided set of 128-token tiles.
//   Q tile  -> shared memory by TMA (4-stage ring) -> TMEM as the A operand (fp16 [128 x hd], converted from bf16 in registers)
//   step n  (64 hidden units):  Aq = Q W1[:, n], Bq = Q W3[:, n]   MMA 128 x 64 x hd, B = weights (K-major)
//            epilogue  Hq = SiLU(Aq) o Bq -> fp16 -> TMEM over its own fp32 source
//            O += Hq W2[n, :]                                      MMA 128 x hd x 64, B = W2 slice (MN-major)
//   O (fp32, TMEM) -> bf16 -> swizzled shared memory -> TMA store (rows beyond M are clipped).
// The fp16 weights of the head (3 x H x hd) sit in shared memory for the CTA's lifetime (TMA, 128-B
// swizzle). Forward accumulators, Q operands and O accumulators are double-buffered in TMEM, so the
// MMA of step n+1 overlaps the SwiGLU epilogue of step n, and Q loads / O stores overlap both.
//
// Warp roles (512 threads): warp 0 = TMA producer (weights once, then Q tiles), warp 1 = MMA issuer,
// warps 4-7 / 8-11 = two epilogue warpgroups alternating steps, warps 12-15 = I/O warpgroup
// (Q: shared -> TMEM; O: TMEM -> shared -> TMA store).
#include <stdio.h>

#include "tc_common.cuh"
#include "ttt_internal.h"

namespace ttt {

int make_token_map(ttt_ctx* ctx, CUtensorMap* map, const void* base, int64_t rows, int64_t cols,
                   int64_t ld, int box_rows);  // bf16_update.cu

namespace app {
constexpr int TM = 128;        // tokens per tile (MMA M)
constexpr int NS = 64;         // hidden units per step
constexpr int THREADS = 896;    // 4 control warps, 16 epilogue warps, 4 O-store warps, 4 Q-load warps
constexpr int IO_WARP0 = 20;    // O: TMEM -> shared -> TMA store
constexpr int QL_WARP0 = 24;    // Q: shared -> TMEM (A operand)
constexpr int QST = 4;         // Q tile ring stages
constexpr int TILE_BYTES = TM * 128;   // one [128 x 64] bf16 tile
// TMEM column plan for hd = 64
constexpr uint32_t C_Q = 0;      // 2 x 32 cols: Q operand (fp16)
constexpr uint32_t C_O = 64;     // 64 cols: O accumulator (fp32), single
constexpr uint32_t C_F = 128;    // 3 x 128 cols: Aq (64) | Bq (64) forward accumulators (fp32)
constexpr int NF = 3;            // forward buffers: two in the epilogue (one per warpgroup) + one in the MMAs
}  // namespace app

__global__ void __launch_bounds__(app::THREADS, 1)
bf16_apply_kernel(const __grid_constant__ CUtensorMap mapW, const __grid_constant__ CUtensorMap mapQ,
                  const __grid_constant__ CUtensorMap mapO, int nh, int H, int tiles_total, int q_early) {
  using namespace app;
  constexpr int HD = 64;
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  // 1024-B aligned base, computed on the 32-bit shared-space address (a uniform value)
  const uint32_t sbase = (smem_u32(smem_raw) + 1023u) & ~1023u;
  uint8_t* smem = smem_raw + (sbase - smem_u32(smem_raw));
  __shared__ uint64_t w_full[8], fwd_full[NF], epi_done[NF], q_full[2], q_empty[2], o_full, o_empty;
  __shared__ uint64_t qr_full[QST], qr_empty[QST];
  __shared__ uint32_t tmem_base_s;

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int h = blockIdx.y;
  const int nsl = H / NS;                                    // steps per tile
  // tiles of this CTA: blockIdx.x, blockIdx.x + gridDim.x, ...
  const int my_tiles = (tiles_total - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
  const int total_steps = my_tiles * nsl;
  const uint32_t w_bytes = 3u * H * 128u;                    // fp16 weights of the head
  uint8_t* q_ring = smem + w_bytes;                          // QST x 16 KB
  uint8_t* o_stage = q_ring + QST * TILE_BYTES;              // 2 x 16 KB

  // Prologue spread over three threads (barriers of the Q ring + first Q requests | other barriers |
  // TMEM allocation). With `q_early` (set by ttt_chunk_step, where the preceding kernels in the
  // stream are this library's own and Q was complete before the first of them started) the first Q
  // tiles are requested BEFORE griddepcontrol.wait, so the first TMA round trip (~2 us with the
  // descriptor fetch) overlaps the tail of the kernel that produces the weights.
  const int npre = min(my_tiles, QST);
  if (tid == 0) {
    tma_prefetch_desc(&mapQ);
    tma_prefetch_desc(&mapW);
    for (int s = 0; s < QST; ++s) mbar_init(&qr_full[s], 1);
    fence_mbar_init();
    if (q_early)
      for (int tl = 0; tl < npre; ++tl) {
        mbar_arrive_expect_tx(&qr_full[tl], TILE_BYTES);
        tma_load_2d_hint(q_ring + tl * TILE_BYTES, &mapQ, &qr_full[tl], h * HD,
                         ((int)blockIdx.x + tl * (int)gridDim.x) * TM, kEvictFirst);
      }
  } else if (tid == 32) {
    for (int n = 0; n < 8; ++n) mbar_init(&w_full[n], 1);
    for (int b = 0; b < NF; ++b) { mbar_init(&fwd_full[b], 1); mbar_init(&epi_done[b], 8); }
    for (int b = 0; b < 2; ++b) { mbar_init(&q_full[b], 128); mbar_init(&q_empty[b], 1); }
    mbar_init(&o_full, 1);
    mbar_init(&o_empty, 128);
    for (int s = 0; s < QST; ++s) mbar_init(&qr_empty[s], 128);
    fence_mbar_init();
  }
  if (warp == 2) { tmem_alloc(&tmem_base_s, 512); tmem_relinquish(); }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  // programmatic dependent launch: everything above overlapped the tail of the preceding kernel
  // (the commit that produces the weights); nothing below may run before it has completed
  asm volatile("griddepcontrol.wait;" ::: "memory");
  const uint32_t tb = tmem_base_s;
  if (tb != 0) __trap();      // all 512 columns belong to this CTA: the issuer uses absolute columns

  if (warp == 0) {
    // ===================== TMA producer: weights once, then the Q tiles =====================
    if (elect_one() && my_tiles > 0) {
      // first Q tile first (it feeds the Q-load warpgroup's shared -> TMEM copy), then the weights step
      // by step, each step on its own barrier so the MMAs start when step 0 has landed
      auto q_load = [&](int tl) {
        mbar_arrive_expect_tx(&qr_full[tl], TILE_BYTES);
        tma_load_2d_hint(q_ring + tl * TILE_BYTES, &mapQ, &qr_full[tl], h * HD,
                         ((int)blockIdx.x + tl * (int)gridDim.x) * TM, kEvictFirst);
      };
      if (!q_early) q_load(0);
      // smem, boxes of 64 rows (8 KB): per 64-hidden step n [W1^T rows | W3^T rows] back to back
      // (one 128-row K-major B operand), then the W2 row blocks
      for (int n = 0; n < nsl; ++n) {
        mbar_arrive_expect_tx(&w_full[n], 3u * 8192u);
        tma_load_2d_hint(smem + (size_t)n * 16384, &mapW, &w_full[n], 0, (0 * nh + h) * H + 64 * n, kEvictLast);
        tma_load_2d_hint(smem + (size_t)n * 16384 + 8192, &mapW, &w_full[n], 0, (2 * nh + h) * H + 64 * n, kEvictLast);
        tma_load_2d_hint(smem + (size_t)nsl * 16384 + (size_t)n * 8192, &mapW, &w_full[n], 0,
                         (1 * nh + h) * H + 64 * n, kEvictLast);
      }
      if (!q_early)
        for (int tl = 1; tl < npre; ++tl) q_load(tl);
      for (int tl = npre; tl < my_tiles; ++tl) {
        const int rs = tl % QST, it = tl / QST;
        mbar_wait(&qr_empty[rs], (it & 1) ^ 1);
        mbar_arrive_expect_tx(&qr_full[rs], TILE_BYTES);
        tma_load_2d_hint(q_ring + rs * TILE_BYTES, &mapQ, &qr_full[rs], h * HD,
                         ((int)blockIdx.x + tl * (int)gridDim.x) * TM, kEvictFirst);
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer =====================
    if (elect_one() && my_tiles > 0) {
      // The issuing thread is bound by its own serial instruction stream: absolute TMEM columns,
      // descriptors that advance by fixed steps, and one 128-wide forward MMA per K step
      // (Aq | Bq in one accumulator: W1^T and W3^T rows of a step are adjacent in shared memory).
      constexpr uint32_t idesc_f = umma_idesc(TM, 2 * NS, 0, 0, TTT_FMT_F16, TTT_FMT_F16);  // A = Q (fp16 in TMEM), B = [W1^T ; W3^T] rows, K-major
      constexpr uint32_t idesc_d = umma_idesc(TM, HD, 0, 1, TTT_FMT_F16, TTT_FMT_F16);      // A = Hq (fp16), B = W2 rows, MN-major
      const uint64_t d13 = umma_smem_desc_sw128(sbase, 16, 1024);
      const uint64_t d2 = umma_smem_desc_sw128(sbase + nsl * 16384, 8192, 1024);
      // forward of step st+1 is issued before the down projection of step st
      int f_tl = 0, f_n = 0;     // (tile, step) of the next forward
      int d_tl = 0, d_n = 0;     // (tile, step) of the next down projection
      int f_fb = 0, d_fb = 0;    // forward buffer (st % NF) and its phase bit (st / NF) & 1
      uint32_t f_ph = 0, d_ph = 0;
      auto fwd = [&]() {
        const int qb = f_tl & 1;
        if (f_n == 0) { mbar_wait(&q_full[qb], (f_tl >> 1) & 1); tc_fence_after(); }
        if (f_tl == 0) { mbar_wait(&w_full[f_n], 0); tc_fence_after(); }     // this step's weights have landed
        const uint32_t acc = C_F + f_fb * 128, qop = C_Q + qb * 32;
        const uint64_t b = d13 + (uint64_t)f_n * 1024;                 // 16 KB per step
#pragma unroll
        for (int k = 0; k < HD / 16; ++k) umma_ts(acc, qop + 8 * k, b + 2 * k, idesc_f, k > 0);
        tc_commit(&fwd_full[f_fb]);
        if (++f_n == nsl) { tc_commit(&q_empty[qb]); f_n = 0; ++f_tl; }
        if (++f_fb == NF) { f_fb = 0; f_ph ^= 1; }
      };
      auto down = [&]() {
        const uint32_t ok = mbar_try_wait(&epi_done[d_fb], d_ph);
        if (d_n == 0 && d_tl > 0) mbar_wait(&o_empty, (d_tl - 1) & 1);   // O of the previous tile is in registers
        if (!ok) mbar_wait(&epi_done[d_fb], d_ph);
        tc_fence_after();
        const uint32_t hq = C_F + d_fb * 128;
        const uint64_t b = d2 + (uint64_t)d_n * 512;                   // 8 KB per step
#pragma unroll
        for (int k = 0; k < NS / 16; ++k)        // Hq K steps 0,1 at columns 0-15, K steps 2,3 at columns 32-47
          umma_ts(C_O, hq + 32 * (k >> 1) + 8 * (k & 1), b + 128 * k, idesc_d, (d_n > 0 || k > 0));
        if (++d_n == nsl) { tc_commit(&o_full); d_n = 0; ++d_tl; }
        if (++d_fb == NF) { d_fb = 0; d_ph ^= 1; }
      };
      // the forward MMAs run two steps ahead of the down projection: one buffer per warpgroup in
      // the epilogue, the third being filled
      fwd();
      if (total_steps > 1) fwd();
      for (int st = 0; st < total_steps; ++st) {
        if (st + 2 < total_steps) fwd();
        down();
      }
    }
  } else if (warp >= 4 && warp < IO_WARP0) {
    // ===================== SwiGLU epilogue warpgroups =====================
    // The two warpgroups alternate steps (three forward buffers keep both fed), so one warpgroup's
    // TMEM load/store phases overlap the other's MUFU burst — the MUFU pipe is the bound of this
    // kernel at hd = 64 (one tanh per element: 512 clk per 128 x 64 step at 16/clk against 384 clk
    // of tensor work).
    // Four warpgroups: pair (wgp & 1) serves the steps of that parity, half (wgp >> 1) owns 32 of
    // the step's 64 hidden columns — four epilogue warps per scheduler, two per step in flight.
    const int wgp = (warp - 4) >> 2, q = warp & 3;
    const int par = wgp & 1, half = wgp >> 1;
    const uint32_t lane_base = static_cast<uint32_t>(q * 32) << 16;
    const uint64_t HALF2 = pack2(0.5f, 0.5f);
    for (int st = par; st < total_steps; st += 2) {
      const int fb = st % NF;
      const uint32_t buf = lane_base + C_F + fb * 128 + 32 * half;   // Aq columns; Bq 64 further
      mbar_wait(&fwd_full[fb], (st / NF) & 1);
      tc_fence_after();
#pragma unroll
      for (int part = 0; part < 2; ++part) {     // 16 hidden columns at a time
        uint32_t ra[16], rb[16];
        tmem_ld_x16(buf + 16 * part, ra);
        tmem_ld_x16(buf + 64 + 16 * part, rb);
        tc_wait_ld();
        uint32_t ph[8];
#pragma unroll
        for (int c = 0; c < 16; c += 2) {
          const uint64_t hf = fmul2(pack2u(ra[c], ra[c + 1]), HALF2);   // a / 2
          const uint64_t bb = pack2u(rb[c], rb[c + 1]);
          float x0, x1;
          unpack2(hf, x0, x1);
          const uint64_t th = pack2(tanh_approx(x0), tanh_approx(x1));
          ph[c >> 1] = pack_f16x2_from2(fmul2(ffma2(hf, th, hf), bb));  // Hq = SiLU(a) b, SiLU(a) = h + h tanh(h)
        }
        tmem_st_x8(buf + 8 * part, ph);          // Hq (fp16) over Aq columns this thread has already read
      }
      tc_wait_st();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&epi_done[fb]);
    }
  } else if (warp >= IO_WARP0) {
    // ===================== I/O warpgroup =====================
    const int q = warp & 3;
    const int r = q * 32 + lane;                               // token row within the tile
    const uint32_t lane_base = static_cast<uint32_t>(q * 32) << 16;
    const uint32_t swz = static_cast<uint32_t>(r & 7);         // 128-B swizzle: chunk ^= row & 7
    auto load_q = [&](int tl) {
      const int qb = tl & 1, rs = tl % QST;
      mbar_wait(&qr_full[rs], (tl / QST) & 1);
      const uint8_t* rowp = q_ring + rs * TILE_BYTES + r * 128;
      uint32_t w[32];
#pragma unroll
      for (int c = 0; c < 8; ++c) {
        const uint4 x = *reinterpret_cast<const uint4*>(rowp + ((c ^ swz) << 4));
        // bf16 -> fp16 on the way to TMEM: every MMA operand is fp16 (ttt_internal.h)
        w[4 * c] = bf16x2_to_f16x2(x.x); w[4 * c + 1] = bf16x2_to_f16x2(x.y);
        w[4 * c + 2] = bf16x2_to_f16x2(x.z); w[4 * c + 3] = bf16x2_to_f16x2(x.w);
      }
      mbar_arrive(&qr_empty[rs]);
      mbar_wait(&q_empty[qb], ((tl >> 1) & 1) ^ 1);
      tc_fence_after();
      tmem_st_x32(tb + lane_base + C_Q + qb * 32, w);
      tc_wait_st();
      tc_fence_before();
      mbar_arrive(&q_full[qb]);
    };
    auto store_o = [&](int tl) {
      const int ob = tl & 1;                                   // shared-memory staging buffer only
      mbar_wait(&o_full, tl & 1);
      tc_fence_after();
      uint32_t ro[64];
      tmem_ld_x32(tb + lane_base + C_O, *reinterpret_cast<uint32_t(*)[32]>(&ro[0]));
      tmem_ld_x32(tb + lane_base + C_O + 32, *reinterpret_cast<uint32_t(*)[32]>(&ro[32]));
      tc_wait_ld();
      tc_fence_before();
      mbar_arrive(&o_empty);                                   // the O accumulator is free again
      // staging buffer `ob` was last used by tile tl-2: its TMA store must have read it
      if (tid == IO_WARP0 * 32) tma_store_wait_read<1>();
      asm volatile("bar.sync 2, 128;" ::: "memory");
      uint8_t* rowp = o_stage + ob * TILE_BYTES + r * 128;
#pragma unroll
      for (int c = 0; c < 8; ++c) {
        uint4 x;
        x.x = pack_bf16x2(__uint_as_float(ro[8 * c]), __uint_as_float(ro[8 * c + 1]));
        x.y = pack_bf16x2(__uint_as_float(ro[8 * c + 2]), __uint_as_float(ro[8 * c + 3]));
        x.z = pack_bf16x2(__uint_as_float(ro[8 * c + 4]), __uint_as_float(ro[8 * c + 5]));
        x.w = pack_bf16x2(__uint_as_float(ro[8 * c + 6]), __uint_as_float(ro[8 * c + 7]));
        *reinterpret_cast<uint4*>(rowp + ((c ^ swz) << 4)) = x;
      }
      fence_proxy_async_smem();
      asm volatile("bar.sync 2, 128;" ::: "memory");
      if (tid == IO_WARP0 * 32) {
        tma_store_2d(&mapO, o_stage + ob * TILE_BYTES, h * HD,
                     ((int)blockIdx.x + tl * (int)gridDim.x) * TM);
        tma_store_commit();
      }
    };
    // separate warpgroups for the two directions: the Q copy of tile tl+2 and the O drain of tile
    // tl are both on the issuer's critical path (Q operand double-buffered, O accumulator single)
    if (warp >= QL_WARP0) {
      for (int tl = 0; tl < my_tiles; ++tl) load_q(tl);
    } else {
      for (int tl = 0; tl < my_tiles; ++tl) store_o(tl);
      if (tid == IO_WARP0 * 32) { tma_store_wait<0>(); }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 2) tmem_dealloc(tb, 512);
}

// ------------------------------------------------------------------------------------------------
int bf16_apply(ttt_ctx* ctx, const __nv_bfloat16* Q, __nv_bfloat16* O, int64_t M, int64_t ld,
               cudaStream_t s) {
  const ttt_config& c = ctx->cfg;
  if (c.hd == 128) return bf16_apply_wide_pair(ctx, Q, O, M, ld, s);   // streamed weights, CTA pairs
  const int tiles = (int)((M + app::TM - 1) / app::TM);
  int per_head = ctx->sm_count / c.nh;
  if (per_head < 1) per_head = 1;
  if (per_head > tiles) per_head = tiles;
  CUtensorMap mapW, mapQ, mapO;
  int rc = make_token_map(ctx, &mapW, ctx->Wb, (int64_t)3 * c.nh * c.hidden, c.hd, c.hd, 64);
  if (rc != TTT_OK) return rc;
  rc = make_token_map(ctx, &mapQ, Q, M, (int64_t)c.nh * c.hd, ld, app::TM);
  if (rc != TTT_OK) return rc;
  rc = make_token_map(ctx, &mapO, O, M, (int64_t)c.nh * c.hd, ld, app::TM);
  if (rc != TTT_OK) return rc;
  const size_t smem = (size_t)3 * c.hidden * 128 + (app::QST + 2) * app::TILE_BYTES + 1024;
  if (smem > ctx->attr_smem_apply) {
    TTT_CUDA_TRY(ctx, cudaFuncSetAttribute(bf16_apply_kernel,
                                           cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem),
                 "bf16_apply_kernel smem attr");
    ctx->attr_smem_apply = smem;
  }
  dim3 grid(per_head, c.nh);
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid;
  cfg.blockDim = dim3(app::THREADS);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = s;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  int nh = c.nh, H = c.hidden, ntl = tiles, q_early = ctx->apply_q_early;
  cudaError_t e = cudaLaunchKernelEx(&cfg, bf16_apply_kernel, mapW, mapQ, mapO, nh, H, ntl, q_early);
  if (e != cudaSuccess) return set_error(ctx, TTT_ERR_CUDA, "bf16_apply_kernel launch", e);
  TTT_LAUNCH_CHECK(ctx, "bf16_apply_kernel");
  return TTT_OK;
}

}  // namespace ttt
