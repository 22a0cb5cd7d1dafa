// bf16_large.cu — the TTT hot path for LARGE head dimensions: the shape the paper itself ships, one
// head of hd = d = 1024 with hidden H = k hd, k in {1, 2, 4} (PAPER.md:382 after Eq. 13; Table 3,
// PAPER.md:242), and in general hd a multiple of 256, H a multiple of 128.
//
// With hd >= 256 nothing of a (head, hidden-slice) fits on one SM any more: the three fp32 gradient
// slices [128 x hd] alone exceed TMEM, and a hidden slice of the weights exceeds shared memory. On the
// other hand every contraction now has all three dimensions >= 256, and the flop-per-byte ratio of the
// layer (~ hd) lets the hidden activations go through HBM once. So the path is four tiled GEMMs, all
// tcgen05 bf16 x bf16 -> fp32 with TMA-fed shared-memory operands and persistent CTAs:
//   update  (Eq. 8 with Eq. 9, Eq. 12)
//     F_u   x | b = K [W1 | W3] and g0 = V W2^T per [128 tokens x 128 hidden] tile (contraction over hd in
//           64-wide chunks), fused SwiGLU forward + backward epilogue -> dA, dB, Hd' = -eta Hd (bf16, HBM)
//     G     G1^T = dA^T K, G3^T = dB^T K, G2 = Hd'^T V per [128 hidden x 256 hd] tile (contraction over ALL
//           tokens of the chunk, both operands MN-major), dense fp32 gradient out (+= pending)
//     commit_plain_kernel (state_kernels.cu): W <- W - G
//   apply   (Eq. 4)
//     F_a   x | b = Q [W1 | W3], epilogue Hq = SiLU(x) b (bf16, HBM)
//     D     O = Hq W2 per [128 tokens x 256 hd] tile (contraction over H, B = W2 rows MN-major)
// Operands are bf16 on this path (weights: the bf16 copy Wq; activations: bf16 keeps fp32's range, so the
// gradient operands need no learning-rate scaling); Newton-Schulz / re-normalisation are not offered
// here (the paper defines neither; ttt_create rejects them for hd > 128).
#include <stdio.h>

#include "tc_common.cuh"
#include "ttt_internal.h"

namespace ttt {

int make_token_map(ttt_ctx* ctx, CUtensorMap* map, const void* base, int64_t rows, int64_t cols,
                   int64_t ld, int box_rows);  // bf16_update.cu

namespace lg {
constexpr int TM = 128;            // rows of an output tile = TMEM lanes
constexpr int KC = 64;             // contraction chunk (one 128-byte swizzled row of bf16)
constexpr int THREADS = 384;       // warp 0 TMA, warp 1 MMA, warp 2 TMEM alloc, warp 3 idle, warps 4-11 epilogue
constexpr int EPI_WARPS = 8;
constexpr int BOX = TM * 128;      // bytes of a [128 rows x 64] bf16 box (16 KB); a [64 x 64] box is BOX / 2
// forward kernels: stage = token chunk + weight-row chunks, 48 KB: [K or Q | W1 | W3] for x | b, or
// [V | W2 | -] for g0. The update runs the two contractions one after the other through the SAME ring
// (a stage holding all five boxes is 80 KB: only two fit, and the TMA round trip was exposed on every
// chunk — 28 K clk per item against 18 K of MMA work)
// plus the epilogue's TMA-store staging tiles (three for the update, one for the apply)
constexpr int F_STAGE = 3 * BOX, F_STAGES_U = 3, F_STAGES_A = 4;
constexpr int F_SMEM_U = F_STAGES_U * F_STAGE + 3 * BOX + 1024, F_SMEM_A = F_STAGES_A * F_STAGE + BOX + 1024;
// CTA-pair variant: a stage is the CTA's token chunk + its HALF of the weight rows = 32 KB
constexpr int P_STAGES_U = 5, P_STAGES_A = 6;
constexpr int P_SMEM_U = P_STAGES_U * 2 * BOX + 3 * BOX + 1024, P_SMEM_A = P_STAGES_A * 2 * BOX + BOX + 1024;
constexpr int P_SMEM_M = 6 * 2 * BOX + 1024;
constexpr uint32_t C_XB = 0, C_G = 256;                // x | b [128 x 256] fp32; g0 [128 x 128] fp32, two buffers
// MN-major-B kernels: stage = A 16 KB + B 32 KB, two accumulators [128 x 256] fp32
constexpr int M_STAGE = 3 * BOX, M_STAGES = 4;
constexpr int TN = 256;
}  // namespace lg

// ------------------------------------------------------------------------------------------------
// F: forward products + SwiGLU epilogue. UPD: update (x | b | g0 -> dA, dB, Hd'); else apply (-> Hq).
// Work item = (token tile tt, hidden slice s, head h), slice fastest; persistent CTAs.
// PAIR: the same on CTA pairs (cluster of 2, tcgen05 cta_group::2, M = 256): a pair takes two adjacent
// token tiles (one per CTA) of a hidden slice and SHARES every B operand — rank 0 loads and holds the
// W1^T rows (x = N columns 0-127) and rows 0-63 of the W2 slice, rank 1 the W3^T rows (b) and W2 rows
// 64-127 — so each CTA streams and reads half of the weight bytes: the single-CTA kernel's SS-mode MMAs
// are bound by the shared-memory pipe (ncu: 57-88 % busy, N = 128 products at 113 clk against 64).
// Rank 0 issues every MMA; both CTAs' TMA loads complete on rank 0's `full` barriers; commits are
// multicast to both CTAs' `empty` / `acc_full`; rank 1's epilogue warps arrive on rank 0's `acc_empty`.
// ------------------------------------------------------------------------------------------------
template <bool UPD, bool LOSS, bool PAIR>
__global__ void __launch_bounds__(lg::THREADS, 1)
ld_forward_kernel(const __grid_constant__ CUtensorMap mapX, const __grid_constant__ CUtensorMap mapV,
                  const __grid_constant__ CUtensorMap mapW, const __grid_constant__ CUtensorMap mapWh,
                  const __grid_constant__ CUtensorMap mapO0,
                  const __grid_constant__ CUtensorMap mapO1, const __grid_constant__ CUtensorMap mapO2,
                  const float* __restrict__ lr, float* __restrict__ loss_part, int M, int nh, int hd,
                  int H, int n_items) {
  using namespace lg;
  constexpr int STAGE = PAIR ? 2 * BOX : F_STAGE;
  constexpr int STAGES = PAIR ? (UPD ? P_STAGES_U : P_STAGES_A) : (UPD ? F_STAGES_U : F_STAGES_A);
  // TMEM: update x | b (256 columns) + two g0 buffers (2 x 128); apply two x | b buffers
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  const uint32_t sbase = (smem_u32(smem_raw) + 1023u) & ~1023u;
  uint8_t* smem = smem_raw + (sbase - smem_u32(smem_raw));
  __shared__ uint64_t full[STAGES], empty[STAGES], acc_full[2], acc_empty[2];
  __shared__ uint32_t tmem_base_s;
  __shared__ float loss_red[EPI_WARPS];

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const uint32_t rank = PAIR ? cluster_rank() : 0u;
  const int cta0 = PAIR ? (int)(blockIdx.x >> 1) : (int)blockIdx.x;     // first item, stride over items
  const int ncta = PAIR ? (int)(gridDim.x >> 1) : (int)gridDim.x;
  const int nslices = H / TM, ntt = (M + TM - 1) / TM, nkc = hd / KC;
  const int ntr = PAIR ? (ntt + 1) / 2 : ntt;                           // token-tile rows of the item space
  if (tid == 0) {
    for (int s = 0; s < STAGES; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], 1); }
    for (int b = 0; b < 2; ++b) { mbar_init(&acc_full[b], 1); mbar_init(&acc_empty[b], (PAIR ? 2 : 1) * EPI_WARPS); }
    fence_mbar_init();
    tma_prefetch_desc(&mapX);
    tma_prefetch_desc(&mapW);
    tma_prefetch_desc(&mapO0);
    if (UPD) tma_prefetch_desc(&mapV);
  }
  if (PAIR) {
    __syncthreads();
    cluster_sync_all();            // the peer's barriers exist before anything can arrive on them
    if (warp == 2) { tmem_alloc2(&tmem_base_s, 512); tmem_relinquish2(); }
  } else {
    if (warp == 2) { tmem_alloc(&tmem_base_s, 512); tmem_relinquish(); }
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tb = tmem_base_s;
  // programmatic dependent launch: the weights (commit) / activations come from the kernel before
  asm volatile("griddepcontrol.wait;" ::: "memory");

  auto item = [&](int id, int& h, int& tt, int& s) {
    s = id % nslices;
    const int r = id / nslices;
    tt = PAIR ? 2 * (r % ntr) + (int)rank : r % ntr;
    h = r / ntr;
  };

  if (warp == 0) {
    // ===================== TMA producer =====================
    if (elect_one()) {
      int g = 0;                                       // running chunk counter over all items
      for (int id = cta0; id < n_items; id += ncta) {
        int h, tt, s;
        item(id, h, tt, s);
        for (int kc = 0; kc < (UPD ? 2 : 1) * nkc; ++kc, ++g) {
          const int st = g % STAGES;
          if (g >= STAGES) mbar_wait(&empty[st], ((g / STAGES) - 1) & 1);
          uint8_t* dst = smem + st * STAGE;
          if (PAIR) {
            const uint32_t bar = mapa_u32(&full[st], 0);           // rank 0's barrier collects both CTAs' bytes
            if (UPD && kc < nkc) {                                 // g0: own V chunk, own half of the W2 rows
              if (rank == 0) mbar_arrive_expect_tx(&full[st], 2 * (BOX + BOX / 2));
              tma_load_2d_pair(dst, &mapV, bar, h * hd + kc * KC, tt * TM);
              tma_load_2d_pair(dst + BOX, &mapWh, bar, kc * KC, (1 * nh + h) * H + s * TM + 64 * (int)rank);
            } else {                                               // x | b: own K / Q chunk, W1^T (rank 0) or W3^T rows
              const int k2 = UPD ? kc - nkc : kc;
              if (rank == 0) mbar_arrive_expect_tx(&full[st], 4 * BOX);
              tma_load_2d_pair(dst, &mapX, bar, h * hd + k2 * KC, tt * TM);
              tma_load_2d_pair(dst + BOX, &mapW, bar, k2 * KC, ((rank ? 2 : 0) * nh + h) * H + s * TM);
            }
            continue;
          }
          if (UPD && kc < nkc) {                         // update, first pass: g0 = V W2^T
            mbar_arrive_expect_tx(&full[st], 2 * BOX);
            tma_load_2d(dst, &mapV, &full[st], h * hd + kc * KC, tt * TM);                            // V chunk
            tma_load_2d(dst + BOX, &mapW, &full[st], kc * KC, (1 * nh + h) * H + s * TM);             // W2 rows
          } else {                                       // x | b = (K or Q) [W1 | W3]
            const int k2 = UPD ? kc - nkc : kc;
            mbar_arrive_expect_tx(&full[st], 3 * BOX);
            tma_load_2d(dst, &mapX, &full[st], h * hd + k2 * KC, tt * TM);                             // K or Q chunk
            tma_load_2d(dst + BOX, &mapW, &full[st], k2 * KC, (0 * nh + h) * H + s * TM);             // W1^T rows
            tma_load_2d(dst + 2 * BOX, &mapW, &full[st], k2 * KC, (2 * nh + h) * H + s * TM);         // W3^T rows
          }
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer =====================
    if (rank == 0 && elect_one()) {
      constexpr uint32_t idesc_xb = umma_idesc_bf16(PAIR ? 2 * TM : TM, 256, 0, 0);   // A = token chunk, B = [W1 ; W3] rows, K-major
      constexpr uint32_t idesc_g = umma_idesc_bf16(PAIR ? 2 * TM : TM, 128, 0, 0);    // A = V chunk, B = W2 rows
      const uint64_t d0 = umma_smem_desc_sw128(sbase, 16, 1024);
      auto mma = [&](uint32_t d, uint64_t a, uint64_t b, uint32_t idesc, uint32_t acc) {
        if (PAIR) umma_ss2(d, a, b, idesc, acc); else umma_ss(d, a, b, idesc, acc);
      };
      auto commit = [&](uint64_t* bar) { if (PAIR) tc_commit2(bar); else tc_commit(bar); };
      int g = 0, n = 0;
      for (int id = cta0; id < n_items; id += ncta, ++n) {
        // update: g0 first, into the g buffer of this item's parity (its last reader, the epilogue of item
        // n - 2, finished before the x | b pass of item n - 1 began), then x | b once the epilogue of item
        // n - 1 has read the previous x | b: that epilogue runs under this item's g0 pass.
        // apply: x | b double-buffered, the epilogue of item n - 2 must have read buffer n & 1.
        const int ab = UPD ? 0 : (n & 1);
        const uint32_t cxb = tb + C_XB + ab * 256, cg = tb + C_G + (n & 1) * 128;
        if (!UPD && n >= 2) { mbar_wait(&acc_empty[ab], ((n >> 1) - 1) & 1); tc_fence_after(); }
        for (int kc = 0; kc < (UPD ? 2 : 1) * nkc; ++kc, ++g) {
          const int st = g % STAGES;
          if (UPD && kc == nkc && n > 0) { mbar_wait(&acc_empty[0], (n - 1) & 1); tc_fence_after(); }
          mbar_wait(&full[st], (g / STAGES) & 1);
          tc_fence_after();
          const uint64_t ds = d0 + (uint64_t)(st * (STAGE >> 4));
          if (UPD && kc < nkc) {
#pragma unroll
            for (int k = 0; k < KC / 16; ++k)
              mma(cg, ds + 2 * k, ds + (BOX >> 4) + 2 * k, idesc_g, (kc > 0) | k);
          } else {
#pragma unroll
            for (int k = 0; k < KC / 16; ++k)
              mma(cxb, ds + 2 * k, ds + (BOX >> 4) + 2 * k, idesc_xb, (kc > (UPD ? nkc : 0)) | k);
          }
          commit(&empty[st]);
        }
        commit(&acc_full[ab]);
      }
    }
  } else if (warp >= 4) {
    // ===================== epilogue: thread = token row (TMEM lane) =====================
    // The 128 hidden columns of the tile go out in two phases of 64 (one 128-byte row of bf16 per token):
    // all eight warps work on a phase (32 rows x 32 columns each), write their operands into swizzled
    // staging tiles [128 rows x 128 B] and one thread hands those to the TMA (a row-per-lane global store
    // touches 32 sectors per instruction and kept the LSU busy for ~6 K clk per tile).
    const int q = warp & 3, half = (warp - 4) >> 2;
    const uint32_t lane_base = static_cast<uint32_t>(q * 32) << 16;
    const uint64_t HALF2 = pack2(0.5f, 0.5f), ONE2 = pack2(1.0f, 1.0f), NONE2 = pack2(-1.0f, -1.0f);
    const int r = q * 32 + lane;                                  // row within the tile
    uint8_t* stg = smem + STAGES * STAGE;                         // NOPS staging tiles of BOX bytes
    const bool leader = tid == 4 * 32;
    int n = 0;
    for (int id = cta0; id < n_items; id += ncta, ++n) {
      int h, tt, s;
      item(id, h, tt, s);
      const int ab = UPD ? 0 : (n & 1);
      const int tok = tt * TM + r;
      float nef = 0.f;
      if (UPD && tok < M) nef = -__ldg(lr + (size_t)h * M + tok);
      const uint64_t ne = pack2(nef, nef);
      uint64_t loss2 = 0ull;
      mbar_wait(&acc_full[ab], (UPD ? n : (n >> 1)) & 1);
      tc_fence_after();
      const uint32_t cxb = tb + lane_base + C_XB + ab * 256, cg = tb + lane_base + C_G + (n & 1) * 128;
#pragma unroll 1
      for (int p = 0; p < 2; ++p) {
        // the staging tiles were handed to the TMA one phase ago: wait until it has read them
        if (leader) tma_store_wait_read<0>();
        asm volatile("bar.sync 1, 256;" ::: "memory");
#pragma unroll 1
        for (int gi = 0; gi < 2; ++gi) {
          const int cl = 2 * half + gi;                           // 16-column group within the phase's 64
          const int c = 4 * p + cl;                               // ... within the tile's 128
          uint32_t rx[16], rb[16], rg[16];
          tmem_ld_x16(cxb + 16 * c, rx);
          tmem_ld_x16(cxb + 128 + 16 * c, rb);
          if (UPD) tmem_ld_x16(cg + 16 * c, rg);
          tc_wait_ld();
          if (p == 1 && gi == 1) {                                // last TMEM read of this tile: release it
            tc_fence_before();
            __syncwarp();
            if (lane == 0) {
              if (rank == 0) mbar_arrive(&acc_empty[ab]); else mbar_arrive_remote(&acc_empty[ab], 0);
            }
          }
          uint32_t pa[8], pb[8], ph[8];
#pragma unroll
          for (int e = 0; e < 16; e += 2) {
            const uint64_t x = fmul2(pack2u(rx[e], rx[e + 1]), HALF2);            // a / 2
            const uint64_t bb = pack2u(rb[e], rb[e + 1]);
            float x0, x1;
            unpack2(x, x0, x1);
            const uint64_t th = pack2(tanh_approx(x0), tanh_approx(x1));
            const uint64_t S = ffma2(x, th, x);                                   // SiLU(a) = a sigmoid(a)
            const uint64_t hdv = fmul2(S, bb);                                    // Hd (update) / Hq (apply)
            if (UPD) {
              const uint64_t g = fmul2(ne, pack2u(rg[e], rg[e + 1]));             // dHd = (-eta v) W2^T
              const uint64_t pp = fadd2(th, ONE2);                                // 2 sigmoid(a)
              const uint64_t m = ffma2(th, NONE2, ONE2);                          // 2 (1 - sigmoid(a))
              const uint64_t t1 = fmul2(ffma2(S, m, pp), HALF2);                  // SiLU'(a)
              pa[e >> 1] = pack_bf16x2_from2(fmul2(fmul2(g, bb), t1));            // dA
              pb[e >> 1] = pack_bf16x2_from2(fmul2(g, S));                        // dB
              ph[e >> 1] = pack_bf16x2_from2(fmul2(ne, hdv));                     // Hd' = -eta Hd
              if (LOSS) loss2 = ffma2(hdv, g, loss2);
            } else {
              ph[e >> 1] = pack_bf16x2_from2(hdv);
            }
          }
          // 16 columns = two 16-byte chunks of the row; 128-byte swizzle: chunk ^= row & 7
          const uint32_t o0 = r * 128 + (((2 * cl) ^ (r & 7)) << 4), o1 = r * 128 + (((2 * cl + 1) ^ (r & 7)) << 4);
          if (UPD) {
            *reinterpret_cast<uint4*>(stg + o0) = make_uint4(pa[0], pa[1], pa[2], pa[3]);
            *reinterpret_cast<uint4*>(stg + o1) = make_uint4(pa[4], pa[5], pa[6], pa[7]);
            *reinterpret_cast<uint4*>(stg + BOX + o0) = make_uint4(pb[0], pb[1], pb[2], pb[3]);
            *reinterpret_cast<uint4*>(stg + BOX + o1) = make_uint4(pb[4], pb[5], pb[6], pb[7]);
          }
          uint8_t* sh = stg + (UPD ? 2 * BOX : 0);
          *reinterpret_cast<uint4*>(sh + o0) = make_uint4(ph[0], ph[1], ph[2], ph[3]);
          *reinterpret_cast<uint4*>(sh + o1) = make_uint4(ph[4], ph[5], ph[6], ph[7]);
        }
        fence_proxy_async_smem();
        asm volatile("bar.sync 1, 256;" ::: "memory");
        if (leader) {                                             // rows beyond M are clipped by the tensor map
          const int col = h * H + s * TM + 64 * p, row = tt * TM;
          if (UPD) {
            tma_store_2d(&mapO0, stg, col, row);
            tma_store_2d(&mapO1, stg + BOX, col, row);
            tma_store_2d(&mapO2, stg + 2 * BOX, col, row);
          } else {
            tma_store_2d(&mapO0, stg, col, row);
          }
          tma_store_commit();
        }
      }
      if (UPD && LOSS) {
        float l0, l1;
        unpack2(loss2, l0, l1);
        float loss = l0 + l1;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) loss += __shfl_xor_sync(0xffffffffu, loss, o);
        if (lane == 0) loss_red[warp - 4] = loss;                // (read two barriers ago at the latest)
        asm volatile("bar.sync 1, 256;" ::: "memory");
        if (leader) {
          float t = 0.f;
          for (int w = 0; w < EPI_WARPS; ++w) t += loss_red[w];
          if (tt < ntt) loss_part[(size_t)(tt * nslices + s) * nh + h] = t;
        }
      }
    }
    if (leader) tma_store_wait<0>();                              // the activations are complete in global memory
  }
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  tc_fence_before();
  __syncthreads();
  if (PAIR) {
    cluster_sync_all();            // neither CTA may leave while the pair's MMAs / remote arrivals can still touch it
    if (warp == 2) tmem_dealloc2(tb, 512);
  } else {
    if (warp == 2) tmem_dealloc(tb, 512);
  }
}

// ------------------------------------------------------------------------------------------------
// G / D: D [128 x 256] (+)= A . B with B MN-major ([contraction rows][256 output columns] in memory).
//   GRAD (A_MN):  tile (matrix j, hidden block hb, hd block nb, head h), contraction over the chunk's tokens;
//                 A = act_j [tokens][hidden] (MN-major), B = K (j = 0, 2) or V (j = 1) [tokens][hd];
//                 out: G[j][h][hb 128 + row][nb 256 + col] (+= when `accumulate`)
//   DOWN:         tile (token tile tt, hd block nb, head h), contraction over H;
//                 A = Hq [tokens][hidden] (K-major), B = W2 rows [hidden][hd]; out: O bf16
// Accumulators are double-buffered in TMEM: the epilogue of a tile overlaps the next tile's main loop.
// PAIR: CTA pairs (cta_group::2, M = 256) as in the forward kernel: two adjacent row blocks (hidden blocks /
// token tiles) share the B operand, rank r loading output columns 128 r .. 128 r + 127 of it (ncu, single
// CTAs: shared-memory pipe 92 % busy in the gradient GEMM).
// ------------------------------------------------------------------------------------------------
template <bool GRAD, bool PAIR>
__global__ void __launch_bounds__(lg::THREADS, 1)
ld_mn_gemm_kernel(const __grid_constant__ CUtensorMap mapA0, const __grid_constant__ CUtensorMap mapA1,
                  const __grid_constant__ CUtensorMap mapA2, const __grid_constant__ CUtensorMap mapB0,
                  const __grid_constant__ CUtensorMap mapB1, float* __restrict__ G,
                  __nv_bfloat16* __restrict__ O, int64_t ldo, int M, int nh, int hd, int H, int n_items,
                  int accumulate) {
  using namespace lg;
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  const uint32_t sbase = (smem_u32(smem_raw) + 1023u) & ~1023u;
  uint8_t* smem = smem_raw + (sbase - smem_u32(smem_raw));
  constexpr int STAGE = PAIR ? 2 * BOX : M_STAGE;           // pairs: A 16 KB + the CTA's half of B 16 KB
  constexpr int STAGES = PAIR ? 6 : M_STAGES;
  __shared__ uint64_t full[STAGES], empty[STAGES], acc_full[2], acc_empty[2];
  __shared__ uint32_t tmem_base_s;

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const uint32_t rank = PAIR ? cluster_rank() : 0u;
  const int cta0 = PAIR ? (int)(blockIdx.x >> 1) : (int)blockIdx.x;
  const int ncta = PAIR ? (int)(gridDim.x >> 1) : (int)gridDim.x;
  const int nnb = hd / TN;                                  // hd blocks of 256
  const int nhb = H / TM, ntt = (M + TM - 1) / TM;
  const int nrb = GRAD ? nhb : ntt;                         // row blocks; pairs take two adjacent ones
  const int nrr = PAIR ? (nrb + 1) / 2 : nrb;
  const int nkc = GRAD ? (M + KC - 1) / KC : H / KC;
  if (tid == 0) {
    for (int s = 0; s < STAGES; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], 1); }
    for (int b = 0; b < 2; ++b) { mbar_init(&acc_full[b], 1); mbar_init(&acc_empty[b], (PAIR ? 2 : 1) * EPI_WARPS); }
    fence_mbar_init();
    tma_prefetch_desc(&mapA0);
    tma_prefetch_desc(&mapB0);
  }
  if (PAIR) {
    __syncthreads();
    cluster_sync_all();
    if (warp == 2) { tmem_alloc2(&tmem_base_s, 512); tmem_relinquish2(); }
  } else {
    if (warp == 2) { tmem_alloc(&tmem_base_s, 512); tmem_relinquish(); }
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tb = tmem_base_s;
  asm volatile("griddepcontrol.wait;" ::: "memory");

  // GRAD: id -> (j, h, hb, nb), nb fastest (the four hd blocks of a hidden block share their A stream);
  // DOWN: id -> (h, tt, nb). A pair's rank 1 may get a row block one past the end (odd count): it runs the
  // MMAs with whatever the loads return and stores nothing.
  auto item = [&](int id, int& j, int& h, int& rb, int& nb) {
    nb = id % nnb;
    int r = id / nnb;
    rb = PAIR ? 2 * (r % nrr) + (int)rank : r % nrr;
    r /= nrr;
    if (GRAD) { h = r % nh; j = r / nh; }
    else { h = r; j = 0; }
  };

  if (warp == 0) {
    if (elect_one()) {
      int g = 0;
      for (int id = cta0; id < n_items; id += ncta) {
        int j, h, rb, nb;
        item(id, j, h, rb, nb);
        const CUtensorMap* mA = GRAD ? (j == 0 ? &mapA0 : j == 1 ? &mapA2 : &mapA1) : &mapA0;   // dA, Hd', dB
        const CUtensorMap* mB = GRAD ? (j == 1 ? &mapB1 : &mapB0) : &mapB0;                      // K | V ; W2 rows
        for (int kc = 0; kc < nkc; ++kc, ++g) {
          const int st = g % STAGES;
          if (g >= STAGES) mbar_wait(&empty[st], ((g / STAGES) - 1) & 1);
          uint8_t* dst = smem + st * STAGE;
          if (PAIR) {
            const uint32_t bar = mapa_u32(&full[st], 0);
            if (rank == 0) mbar_arrive_expect_tx(&full[st], 4 * BOX);
            if (GRAD) {
              tma_load_2d_pair(dst, mA, bar, h * H + rb * TM, kc * KC);
              tma_load_2d_pair(dst + BOX / 2, mA, bar, h * H + rb * TM + 64, kc * KC);
              for (int a = 0; a < 2; ++a)               // this CTA's two of the four hd atoms
                tma_load_2d_pair(dst + BOX + a * (BOX / 2), mB, bar, h * hd + nb * TN + 128 * (int)rank + 64 * a, kc * KC);
            } else {
              tma_load_2d_pair(dst, mA, bar, h * H + kc * KC, rb * TM);
              for (int a = 0; a < 2; ++a)
                tma_load_2d_pair(dst + BOX + a * (BOX / 2), mB, bar, nb * TN + 128 * (int)rank + 64 * a, (1 * nh + h) * H + kc * KC);
            }
            continue;
          }
          mbar_arrive_expect_tx(&full[st], M_STAGE);
          if (GRAD) {
            // A: two [64 tokens x 64 hidden] atoms (hidden halves of the block)
            tma_load_2d(dst, mA, &full[st], h * H + rb * TM, kc * KC);
            tma_load_2d(dst + BOX / 2, mA, &full[st], h * H + rb * TM + 64, kc * KC);
            // B: four [64 tokens x 64 hd] atoms
            for (int a = 0; a < 4; ++a)
              tma_load_2d(dst + BOX + a * (BOX / 2), mB, &full[st], h * hd + nb * TN + 64 * a, kc * KC);
          } else {
            tma_load_2d(dst, mA, &full[st], h * H + kc * KC, rb * TM);              // Hq [128 tokens x 64 hidden]
            for (int a = 0; a < 4; ++a)                                             // W2 rows [64 hidden x 64 hd] x 4
              tma_load_2d(dst + BOX + a * (BOX / 2), mB, &full[st], nb * TN + 64 * a, (1 * nh + h) * H + kc * KC);
          }
        }
      }
    }
  } else if (warp == 1) {
    if (rank == 0 && elect_one()) {
      constexpr uint32_t idesc = umma_idesc_bf16(PAIR ? 2 * TM : TM, TN, GRAD ? 1 : 0, 1);
      const uint64_t dA = GRAD ? umma_smem_desc_sw128(sbase, BOX / 2, 1024) : umma_smem_desc_sw128(sbase, 16, 1024);
      const uint64_t dB = umma_smem_desc_sw128(sbase + BOX, BOX / 2, 1024);
      int g = 0, n = 0;
      for (int id = cta0; id < n_items; id += ncta, ++n) {
        const int ab = n & 1;
        if (n >= 2) { mbar_wait(&acc_empty[ab], ((n >> 1) - 1) & 1); tc_fence_after(); }
        const uint32_t acc = tb + ab * TN;
        for (int kc = 0; kc < nkc; ++kc, ++g) {
          const int st = g % STAGES;
          mbar_wait(&full[st], (g / STAGES) & 1);
          tc_fence_after();
          const uint64_t so = (uint64_t)(st * (STAGE >> 4));
#pragma unroll
          for (int k = 0; k < KC / 16; ++k) {          // MN-major: +2048 B per 16-row K step; K-major: +32 B
            if (PAIR) umma_ss2(acc, dA + so + (GRAD ? 128 * k : 2 * k), dB + so + 128 * k, idesc, (kc > 0) | k);
            else umma_ss(acc, dA + so + (GRAD ? 128 * k : 2 * k), dB + so + 128 * k, idesc, (kc > 0) | k);
          }
          if (PAIR) tc_commit2(&empty[st]); else tc_commit(&empty[st]);
        }
        if (PAIR) tc_commit2(&acc_full[ab]); else tc_commit(&acc_full[ab]);
      }
    }
  } else if (warp >= 4) {
    const int q = warp & 3, half = (warp - 4) >> 2;
    const uint32_t lane_base = static_cast<uint32_t>(q * 32) << 16;
    int n = 0;
    for (int id = cta0; id < n_items; id += ncta, ++n) {
      int j, h, rb, nb;
      item(id, j, h, rb, nb);
      const int ab = n & 1;
      const int row = rb * TM + q * 32 + lane;
      const bool live = rb < nrb;                      // (a pair's rank 1 one past the last row block)
      mbar_wait(&acc_full[ab], (n >> 1) & 1);
      tc_fence_after();
#pragma unroll 1
      for (int c = 0; c < 4; ++c) {                    // 32 columns per TMEM round trip
        uint32_t r[32];
        tmem_ld_x32(tb + lane_base + ab * TN + 128 * half + 32 * c, r);
        tc_wait_ld();
        const int col = nb * TN + 128 * half + 32 * c;
        if (!live) continue;
        if (GRAD) {
          float4* dst = reinterpret_cast<float4*>(G + (((size_t)j * nh + h) * H + row) * hd + col);
#pragma unroll
          for (int v = 0; v < 8; ++v) {
            float4 o = make_float4(__uint_as_float(r[4 * v]), __uint_as_float(r[4 * v + 1]),
                                   __uint_as_float(r[4 * v + 2]), __uint_as_float(r[4 * v + 3]));
            if (accumulate) { const float4 p = dst[v]; o.x += p.x; o.y += p.y; o.z += p.z; o.w += p.w; }
            dst[v] = o;
          }
        } else if (row < M) {
          uint4* dst = reinterpret_cast<uint4*>(O + (size_t)row * ldo + (size_t)h * hd + col);
#pragma unroll
          for (int v = 0; v < 4; ++v)
            dst[v] = make_uint4(pack_bf16x2(__uint_as_float(r[8 * v]), __uint_as_float(r[8 * v + 1])),
                                pack_bf16x2(__uint_as_float(r[8 * v + 2]), __uint_as_float(r[8 * v + 3])),
                                pack_bf16x2(__uint_as_float(r[8 * v + 4]), __uint_as_float(r[8 * v + 5])),
                                pack_bf16x2(__uint_as_float(r[8 * v + 6]), __uint_as_float(r[8 * v + 7])));
        }
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) {
        if (rank == 0) mbar_arrive(&acc_empty[ab]); else mbar_arrive_remote(&acc_empty[ab], 0);
      }
    }
  }
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  tc_fence_before();
  __syncthreads();
  if (PAIR) {
    cluster_sync_all();
    if (warp == 2) tmem_dealloc2(tb, 512);
  } else {
    if (warp == 2) tmem_dealloc(tb, 512);
  }
}

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------
int bf16_large_supported(const ttt_config* cfg) {
  return cfg->act_dtype == TTT_BF16 && cfg->hd >= 256 && cfg->hd % 256 == 0 && cfg->hd <= 2048 &&
         cfg->hidden % 128 == 0 && cfg->ns_iters == 0 && cfg->renorm == 0 && !cfg->linear_fast_weight;
}

int64_t bf16_large_loss_rows(const ttt_config* cfg) {
  return ((cfg->max_tokens + lg::TM - 1) / lg::TM) * (cfg->hidden / lg::TM);
}

// `cluster` = 2 launches CTA pairs (grid = 2 x pairs)
template <typename Kern, typename... Args>
static int launch_pdl(ttt_ctx* ctx, const char* what, Kern kern, int grid, size_t smem, cudaStream_t s, int cluster,
                      Args... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(grid);
  cfg.blockDim = dim3(lg::THREADS);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = s;
  cudaLaunchAttribute attr[2];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  attr[1].id = cudaLaunchAttributeClusterDimension;
  attr[1].val.clusterDim.x = cluster;
  attr[1].val.clusterDim.y = 1;
  attr[1].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = cluster > 1 ? 2 : 1;
  cudaError_t e = cudaLaunchKernelEx(&cfg, kern, args...);
  if (e != cudaSuccess) return set_error(ctx, TTT_ERR_CUDA, what, e);
  e = cudaGetLastError();
  if (e != cudaSuccess) return set_error(ctx, TTT_ERR_CUDA, what, e);
  ctx->launches += 1;
  return TTT_OK;
}

static int large_attrs(ttt_ctx* ctx) {
  if (ctx->attr_done & ATTR_LARGE) return TTT_OK;
  const int su = lg::F_SMEM_U, sa = lg::F_SMEM_A;
  const int sm = lg::M_STAGE * lg::M_STAGES + 1024;
  TTT_CUDA_TRY(ctx, cudaFuncSetAttribute(ld_forward_kernel<true, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, su), "ld_forward smem attr");
  TTT_CUDA_TRY(ctx, cudaFuncSetAttribute(ld_forward_kernel<true, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, su), "ld_forward smem attr");
  TTT_CUDA_TRY(ctx, cudaFuncSetAttribute(ld_forward_kernel<false, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, sa), "ld_forward smem attr");
  TTT_CUDA_TRY(ctx, cudaFuncSetAttribute(ld_forward_kernel<true, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, lg::P_SMEM_U), "ld_forward smem attr");
  TTT_CUDA_TRY(ctx, cudaFuncSetAttribute(ld_forward_kernel<true, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, lg::P_SMEM_U), "ld_forward smem attr");
  TTT_CUDA_TRY(ctx, cudaFuncSetAttribute(ld_forward_kernel<false, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, lg::P_SMEM_A), "ld_forward smem attr");
  {   // CTA pairs the device can host at once (0 -> the single-CTA kernels are used)
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(2 * (ctx->sm_count / 2));
    cfg.blockDim = dim3(lg::THREADS);
    cfg.dynamicSmemBytes = lg::P_SMEM_U;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = 2;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    int n = 0;
    if (cudaOccupancyMaxActiveClusters(&n, ld_forward_kernel<true, false, true>, &cfg) != cudaSuccess) { n = 0; cudaGetLastError(); }
    ctx->ld_pairs = n;
  }
  TTT_CUDA_TRY(ctx, cudaFuncSetAttribute(ld_mn_gemm_kernel<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm), "ld_mn_gemm smem attr");
  TTT_CUDA_TRY(ctx, cudaFuncSetAttribute(ld_mn_gemm_kernel<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm), "ld_mn_gemm smem attr");
  TTT_CUDA_TRY(ctx, cudaFuncSetAttribute(ld_mn_gemm_kernel<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, lg::P_SMEM_M), "ld_mn_gemm smem attr");
  TTT_CUDA_TRY(ctx, cudaFuncSetAttribute(ld_mn_gemm_kernel<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, lg::P_SMEM_M), "ld_mn_gemm smem attr");
  ctx->attr_done |= ATTR_LARGE;
  return TTT_OK;
}

// steps 1-5: forward + epilogue, then the three gradient GEMMs into the dense pending gradient G
int bf16_large_accumulate(ttt_ctx* ctx, const __nv_bfloat16* K, const __nv_bfloat16* V, const float* lr,
                          int64_t M, int64_t ld, bool want_loss, int* loss_rows, cudaStream_t s) {
  const ttt_config& c = ctx->cfg;
  int rc = large_attrs(ctx);
  if (rc != TTT_OK) return rc;
  const int64_t HW = (int64_t)c.nh * c.hidden;
  CUtensorMap mK, mV, mW, mA0, mA1, mA2, mK64, mV64;
  if ((rc = make_token_map(ctx, &mK, K, M, (int64_t)c.nh * c.hd, ld, lg::TM)) != TTT_OK) return rc;
  if ((rc = make_token_map(ctx, &mV, V, M, (int64_t)c.nh * c.hd, ld, lg::TM)) != TTT_OK) return rc;
  if ((rc = make_token_map(ctx, &mW, ctx->Wq, (int64_t)3 * c.nh * c.hidden, c.hd, c.hd, lg::TM)) != TTT_OK) return rc;
  if ((rc = make_token_map(ctx, &mA0, ctx->lact[0], M, HW, HW, 64)) != TTT_OK) return rc;
  if ((rc = make_token_map(ctx, &mA1, ctx->lact[1], M, HW, HW, 64)) != TTT_OK) return rc;
  if ((rc = make_token_map(ctx, &mA2, ctx->lact[2], M, HW, HW, 64)) != TTT_OK) return rc;
  CUtensorMap mS0, mS1, mS2;                      // the forward kernel's TMA stores: boxes of [128 tokens][64]
  if ((rc = make_token_map(ctx, &mS0, ctx->lact[0], M, HW, HW, lg::TM)) != TTT_OK) return rc;
  if ((rc = make_token_map(ctx, &mS1, ctx->lact[1], M, HW, HW, lg::TM)) != TTT_OK) return rc;
  if ((rc = make_token_map(ctx, &mS2, ctx->lact[2], M, HW, HW, lg::TM)) != TTT_OK) return rc;
  if ((rc = make_token_map(ctx, &mK64, K, M, (int64_t)c.nh * c.hd, ld, 64)) != TTT_OK) return rc;
  if ((rc = make_token_map(ctx, &mV64, V, M, (int64_t)c.nh * c.hd, ld, 64)) != TTT_OK) return rc;
  const int ntt = (int)((M + lg::TM - 1) / lg::TM), nsl = c.hidden / lg::TM;
  CUtensorMap mWh;                                 // weight rows in boxes of 64 (a CTA pair's half of the W2 slice)
  if ((rc = make_token_map(ctx, &mWh, ctx->Wq, (int64_t)3 * c.nh * c.hidden, c.hd, c.hd, 64)) != TTT_OK) return rc;
  int n_items = c.nh * ntt * nsl;
  int grid = n_items < ctx->sm_count ? n_items : ctx->sm_count;
  int Mi = (int)M, nh = c.nh, hd = c.hd, H = c.hidden;
  if (ctx->ld_pairs > 0) {
    n_items = c.nh * ((ntt + 1) / 2) * nsl;          // items of a pair: two adjacent token tiles x one slice
    grid = 2 * (n_items < ctx->ld_pairs ? n_items : ctx->ld_pairs);
    if (want_loss)
      rc = launch_pdl(ctx, "ld_forward_kernel (update, pairs)", ld_forward_kernel<true, true, true>, grid, (size_t)lg::P_SMEM_U, s, 2,
                      mK, mV, mW, mWh, mS0, mS1, mS2, lr, ctx->loss_part, Mi, nh, hd, H, n_items);
    else
      rc = launch_pdl(ctx, "ld_forward_kernel (update, pairs)", ld_forward_kernel<true, false, true>, grid, (size_t)lg::P_SMEM_U, s, 2,
                      mK, mV, mW, mWh, mS0, mS1, mS2, lr, ctx->loss_part, Mi, nh, hd, H, n_items);
  } else if (want_loss) {
    rc = launch_pdl(ctx, "ld_forward_kernel (update)", ld_forward_kernel<true, true, false>, grid, (size_t)lg::F_SMEM_U, s, 1,
                    mK, mV, mW, mWh, mS0, mS1, mS2, lr, ctx->loss_part, Mi, nh, hd, H, n_items);
  } else {
    rc = launch_pdl(ctx, "ld_forward_kernel (update)", ld_forward_kernel<true, false, false>, grid, (size_t)lg::F_SMEM_U, s, 1,
                    mK, mV, mW, mWh, mS0, mS1, mS2, lr, ctx->loss_part, Mi, nh, hd, H, n_items);
  }
  if (rc != TTT_OK) return rc;
  *loss_rows = ntt * nsl;
  int accumulate = ctx->G_valid ? 1 : 0;
  __nv_bfloat16* nullo = nullptr;
  int64_t ldo = 0;
  if (ctx->ld_pairs > 0) {
    n_items = 3 * c.nh * ((nsl + 1) / 2) * (c.hd / lg::TN);
    grid = 2 * (n_items < ctx->ld_pairs ? n_items : ctx->ld_pairs);
    rc = launch_pdl(ctx, "ld_mn_gemm_kernel (gradient, pairs)", ld_mn_gemm_kernel<true, true>, grid, (size_t)lg::P_SMEM_M, s, 2,
                    mA0, mA1, mA2, mK64, mV64, ctx->G, nullo, ldo, Mi, nh, hd, H, n_items, accumulate);
  } else {
    n_items = 3 * c.nh * nsl * (c.hd / lg::TN);
    grid = n_items < ctx->sm_count ? n_items : ctx->sm_count;
    rc = launch_pdl(ctx, "ld_mn_gemm_kernel (gradient)", ld_mn_gemm_kernel<true, false>, grid,
                    (size_t)lg::M_STAGE * lg::M_STAGES + 1024, s, 1, mA0, mA1, mA2, mK64, mV64,
                    ctx->G, nullo, ldo, Mi, nh, hd, H, n_items, accumulate);
  }
  if (rc != TTT_OK) return rc;
  ctx->G_valid = true;
  return TTT_OK;
}

int bf16_large_apply(ttt_ctx* ctx, const __nv_bfloat16* Q, __nv_bfloat16* O, int64_t M, int64_t ld,
                     cudaStream_t s) {
  const ttt_config& c = ctx->cfg;
  int rc = large_attrs(ctx);
  if (rc != TTT_OK) return rc;
  const int64_t HW = (int64_t)c.nh * c.hidden;
  CUtensorMap mQ, mW, mHq, mW64;
  if ((rc = make_token_map(ctx, &mQ, Q, M, (int64_t)c.nh * c.hd, ld, lg::TM)) != TTT_OK) return rc;
  if ((rc = make_token_map(ctx, &mW, ctx->Wq, (int64_t)3 * c.nh * c.hidden, c.hd, c.hd, lg::TM)) != TTT_OK) return rc;
  if ((rc = make_token_map(ctx, &mHq, ctx->lact[0], M, HW, HW, lg::TM)) != TTT_OK) return rc;
  if ((rc = make_token_map(ctx, &mW64, ctx->Wq, (int64_t)3 * c.nh * c.hidden, c.hd, c.hd, 64)) != TTT_OK) return rc;
  const int ntt = (int)((M + lg::TM - 1) / lg::TM), nsl = c.hidden / lg::TM;
  int n_items = c.nh * ntt * nsl;
  int grid = n_items < ctx->sm_count ? n_items : ctx->sm_count;
  int Mi = (int)M, nh = c.nh, hd = c.hd, H = c.hidden;
  const float* nolr = nullptr;
  float* nof = nullptr;
  if (ctx->ld_pairs > 0) {
    n_items = c.nh * ((ntt + 1) / 2) * nsl;
    grid = 2 * (n_items < ctx->ld_pairs ? n_items : ctx->ld_pairs);
    rc = launch_pdl(ctx, "ld_forward_kernel (apply, pairs)", ld_forward_kernel<false, false, true>, grid, (size_t)lg::P_SMEM_A, s, 2,
                    mQ, mQ, mW, mW64, mHq, mHq, mHq, nolr, nof, Mi, nh, hd, H, n_items);
  } else {
    rc = launch_pdl(ctx, "ld_forward_kernel (apply)", ld_forward_kernel<false, false, false>, grid, (size_t)lg::F_SMEM_A, s, 1,
                    mQ, mQ, mW, mW64, mHq, mHq, mHq, nolr, nof, Mi, nh, hd, H, n_items);
  }
  if (rc != TTT_OK) return rc;
  int accumulate = 0;
  if (ctx->ld_pairs > 0) {
    n_items = c.nh * ((ntt + 1) / 2) * (c.hd / lg::TN);
    grid = 2 * (n_items < ctx->ld_pairs ? n_items : ctx->ld_pairs);
    return launch_pdl(ctx, "ld_mn_gemm_kernel (down projection, pairs)", ld_mn_gemm_kernel<false, true>, grid,
                      (size_t)lg::P_SMEM_M, s, 2, mHq, mHq, mHq, mW64, mW64, nof, O, ld, Mi, nh, hd, H, n_items, accumulate);
  }
  n_items = c.nh * ntt * (c.hd / lg::TN);
  grid = n_items < ctx->sm_count ? n_items : ctx->sm_count;
  return launch_pdl(ctx, "ld_mn_gemm_kernel (down projection)", ld_mn_gemm_kernel<false, false>, grid,
                    (size_t)lg::M_STAGE * lg::M_STAGES + 1024, s, 1, mHq, mHq, mHq,
                    mW64, mW64, nof, O, ld, Mi, nh, hd, H, n_items, accumulate);
}

}  // namespace ttt
