// ns_tc_wide.cu — Newton-Schulz orthonormalisation on the tensor cores for head dimension 128
// (reading R-NS; BASELINE.json configs[4]: 8 heads x 128, hidden 512).
//
// Tall form of the iteration on X [H x 128] (hidden-major), as in ns_tc.cu:
//     X0 = g / (||g||_F + 1e-7);   n times:  A = X^T X;  Pm = a I + b A + c A A;  X <- X Pm
// with every product as a split-bf16 ("bf16x3") contraction hi*hi + hi*lo + lo*hi, fp32 accumulation.
//
// At hd = 128 the hi / lo operand tiles of a whole matrix (256 KB at H = 512) exceed one SM's shared
// memory, so a matrix is owned by a thread-block cluster of H / 128 CTAs, one 128-row block each:
//   Gram   every CTA forms the partial A_r = X_r^T X_r of its rows (MN-major operands) and writes it as
//          fp32 to a scratch in global memory (L2); after a cluster barrier every CTA sums the partials
//          of all ranks in rank order (so all ranks hold bit-identical A). Distributed shared memory
//          was measured first: ~20 B/clk per SM made the exchange 80 % of the kernel;
//   square A A and Pm are computed redundantly by every rank (128 x 128 x 128, cheap);
//   tall   X_r <- X_r Pm needs no exchange.
// The accumulator layout (TMEM lane = row, 32 columns per warp) is also the register layout of A and
// X, so the folds need no transposition: TMEM -> registers -> hi/lo split -> swizzled operand tiles.
// Global traffic (load, exchange, write-out) is coalesced through one padded fp32 staging tile.
#include <stdio.h>

#include "tc_common.cuh"
#include "ttt_internal.h"

namespace ttt {

namespace nsw {
constexpr int HD = 128;
constexpr int RB = 128;          // rows of X per CTA
constexpr int THREADS = 512;     // fold / load workers (16 warps)
constexpr int LAUNCH_THREADS = THREADS + 32;   // + the MMA-issuing warp (warp 16)
constexpr int SUB = RB * 128;    // one [128 rows x 64] bf16 sub-tile (16 KB)
constexpr int TILE = 2 * SUB;    // one [128 x 128] bf16 operand tile
constexpr int EX_LD = 132;       // fp32 exchange row stride in floats (16-B aligned, conflict-free float4)
constexpr size_t SMEM_BYTES = 4 * (size_t)TILE + (size_t)RB * EX_LD * sizeof(float) + 1024;
constexpr uint32_t C_A = 0, C_A2 = 128, C_X = 256;
}  // namespace nsw

__device__ __forceinline__ uint32_t cluster_ctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ void cluster_arrive() {
  asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
}
__device__ __forceinline__ void cluster_wait() {
  asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ uint32_t dsmem_addr(uint32_t local_addr, uint32_t rank) {
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(local_addr), "r"(rank));
  return r;
}
__device__ __forceinline__ float4 ld_dsmem_f4(uint32_t addr) {
  float4 v;
  asm volatile("ld.shared::cluster.v4.f32 {%0, %1, %2, %3}, [%4];"
               : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr) : "memory");
  return v;
}
__device__ __forceinline__ float ld_dsmem_f(uint32_t addr) {
  float v;
  asm volatile("ld.shared::cluster.f32 %0, [%1];" : "=f"(v) : "r"(addr) : "memory");
  return v;
}

// 32 fp32 values of one row (columns 32 cs .. 32 cs + 31) -> hi / lo bf16 into a [128 x 128] operand
// tile pair stored as two 128-byte-swizzled [128 x 64] sub-tiles
__device__ __forceinline__ void split_row32(const float (&v)[32], uint8_t* hi_tile, uint8_t* lo_tile,
                                            int row, int cs) {
  uint8_t* hs = hi_tile + (cs >> 1) * nsw::SUB;
  uint8_t* ls = lo_tile + (cs >> 1) * nsw::SUB;
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    uint32_t h[4], l[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const float a = v[8 * k + 2 * i], b = v[8 * k + 2 * i + 1];
      h[i] = pack_bf16x2(a, b);
      l[i] = pack_bf16x2(a - __uint_as_float(h[i] << 16), b - __uint_as_float(h[i] & 0xffff0000u));
    }
    const int chunk = (cs & 1) * 4 + k;                    // 16-byte chunk within the 128-byte row
    const uint32_t off = static_cast<uint32_t>(row * 128 + ((chunk ^ (row & 7)) << 4));
    *reinterpret_cast<uint4*>(hs + off) = make_uint4(h[0], h[1], h[2], h[3]);
    *reinterpret_cast<uint4*>(ls + off) = make_uint4(l[0], l[1], l[2], l[3]);
  }
}

__global__ void __launch_bounds__(nsw::LAUNCH_THREADS, 1)
ns_tc_wide_kernel(float* __restrict__ G, const float* __restrict__ P, int n_sets, size_t set_elems,
                  int use_G, int H, int iters, float* __restrict__ Wm, ttt_wop_t* __restrict__ Wb, __nv_bfloat16* __restrict__ Wq,
                  float* __restrict__ scratch) {
  using namespace nsw;
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  const uint32_t sbase = (smem_u32(smem_raw) + 1023u) & ~1023u;
  uint8_t* smem = smem_raw + (sbase - smem_u32(smem_raw));
  uint8_t* XH = smem;
  uint8_t* XL = XH + TILE;
  uint8_t* AH = XL + TILE;             // A, then Pm (hi)
  uint8_t* AL = AH + TILE;
  float* EX = reinterpret_cast<float*>(AL + TILE);          // [128][EX_LD] fp32 staging (row <-> coalesced)
  __shared__ uint64_t mma_bar;
  __shared__ uint32_t tmem_base_s;
  __shared__ float red[THREADS / 32];
  __shared__ float s_part;

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const bool issuer = warp == THREADS / 32;
  const uint32_t rank = cluster_ctarank(), nc = gridDim.x;   // the cluster spans the grid's x dimension
  const int q = warp & 3, cs = (warp >> 2) & 3;              // TMEM lane quarter, 32-column group
  const int trow = q * 32 + lane;                            // row of the block = TMEM lane
  const uint32_t lane_base = static_cast<uint32_t>(q * 32) << 16;
  // this rank's [128 x 128] block of the matrix; float4 index e = tid + 512 k <-> (row e / 32, cols 4 (e % 32))
  const size_t blk = ((size_t)blockIdx.y * H + (size_t)rank * RB) * HD;
  float* ex_row = EX + trow * EX_LD + 32 * cs;               // row layout: this thread's 32 columns
  auto ex_co = [&](int k) { const int e = tid + THREADS * k; return EX + (e >> 5) * EX_LD + (e & 31) * 4; };
  auto worker_bar = [&]() { asm volatile("bar.sync 2, 512;" ::: "memory"); };
  auto rows_to_ex = [&](const float (&v)[32]) {
#pragma unroll
    for (int u = 0; u < 8; ++u)
      reinterpret_cast<float4*>(ex_row)[u] = make_float4(v[4 * u], v[4 * u + 1], v[4 * u + 2], v[4 * u + 3]);
  };
  auto ex_to_rows = [&](float (&v)[32]) {
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      const float4 x = reinterpret_cast<const float4*>(ex_row)[u];
      v[4 * u] = x.x; v[4 * u + 1] = x.y; v[4 * u + 2] = x.z; v[4 * u + 3] = x.w;
    }
  };

  if (tid == 0) { mbar_init(&mma_bar, 1); fence_mbar_init(); }
  if (warp == 0) { tmem_alloc(&tmem_base_s, 512); tmem_relinquish(); }
  // programmatic dependent launch: the set-up above overlapped the tail of the gradient kernel
  asm volatile("griddepcontrol.wait;" ::: "memory");

  // ---- load (coalesced): g = (use_G ? G : 0) + sum_s P[s] (fixed order); Frobenius norm over the cluster ----
  float4 g[8];
  float acc = 0.f;
  if (!issuer) {
#pragma unroll
    for (int k = 0; k < 8; ++k)
      g[k] = use_G ? reinterpret_cast<const float4*>(G + blk)[tid + THREADS * k] : make_float4(0.f, 0.f, 0.f, 0.f);
    for (int s = 0; s < n_sets; s += 2) {              // two sets in flight, summed in set order
      const float4* p0 = reinterpret_cast<const float4*>(P + (size_t)s * set_elems + blk);
      const float4* p1 = reinterpret_cast<const float4*>(P + (size_t)(s + 1) * set_elems + blk);
      const bool two = s + 1 < n_sets;
      float4 a[8], b[8];
#pragma unroll
      for (int k = 0; k < 8; ++k) {
        a[k] = __ldcg(p0 + tid + THREADS * k);
        b[k] = two ? __ldcg(p1 + tid + THREADS * k) : make_float4(0.f, 0.f, 0.f, 0.f);
      }
#pragma unroll
      for (int k = 0; k < 8; ++k) {
        g[k].x = (g[k].x + a[k].x) + b[k].x; g[k].y = (g[k].y + a[k].y) + b[k].y;
        g[k].z = (g[k].z + a[k].z) + b[k].z; g[k].w = (g[k].w + a[k].w) + b[k].w;
      }
    }
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      acc = fmaf(g[k].x, g[k].x, acc); acc = fmaf(g[k].y, g[k].y, acc);
      acc = fmaf(g[k].z, g[k].z, acc); acc = fmaf(g[k].w, g[k].w, acc);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if (lane == 0) red[warp] = acc;
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tb = tmem_base_s;
  if (tid == 0) {
    float t = 0.f;
    for (int w = 0; w < THREADS / 32; ++w) t += red[w];
    s_part = t;
  }
  __syncthreads();
  cluster_arrive();
  cluster_wait();
  float scale;
  {
    float t = 0.f;
    for (uint32_t r = 0; r < nc; ++r) t += ld_dsmem_f(dsmem_addr(smem_u32(&s_part), r));   // rank order
    scale = 1.0f / (sqrtf(t) + 1e-7f);
  }
  if (!issuer) {
#pragma unroll
    for (int k = 0; k < 8; ++k)
      *reinterpret_cast<float4*>(ex_co(k)) = make_float4(g[k].x * scale, g[k].y * scale, g[k].z * scale, g[k].w * scale);
    worker_bar();
    float x[32];
    ex_to_rows(x);
    split_row32(x, XH, XL, trow, cs);
  }
  fence_proxy_async_smem();
  __syncthreads();

  constexpr uint32_t idesc_mn = umma_idesc_bf16(128, 128, 1, 1);   // A, B MN-major (Gram)
  constexpr uint32_t idesc_k = umma_idesc_bf16(128, 128, 0, 0);    // A, B K-major
  const uint64_t d_xh_mn = umma_smem_desc_sw128(smem_u32(XH), SUB, 1024);   // 2nd 64-column atom: +SUB
  const uint64_t d_xl_mn = umma_smem_desc_sw128(smem_u32(XL), SUB, 1024);
  const uint64_t d_xh = umma_smem_desc_sw128(smem_u32(XH), 16, 1024);
  const uint64_t d_xl = umma_smem_desc_sw128(smem_u32(XL), 16, 1024);
  const uint64_t d_ah = umma_smem_desc_sw128(smem_u32(AH), 16, 1024);
  const uint64_t d_al = umma_smem_desc_sw128(smem_u32(AL), 16, 1024);
  const float ca = 3.4445f, cb = -4.7750f, cc = 2.0315f;
  uint32_t phase = 0;
  float Areg[32];
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
  // K-major split product D = (AH + AL) (BH + BL)^T without the lo*lo term, 128 x 128 x 128
  auto product_k = [&](uint32_t dcol, uint64_t ah, uint64_t al, uint64_t bh, uint64_t bl) {
#pragma unroll
    for (int k = 0; k < HD / 16; ++k) {
      const uint64_t o = (uint64_t)((k >> 2) * (SUB >> 4) + (k & 3) * 2);
      umma_ss(dcol, ah + o, bh + o, idesc_k, k > 0);
      umma_ss(dcol, ah + o, bl + o, idesc_k, 1);
      umma_ss(dcol, al + o, bh + o, idesc_k, 1);
    }
    tc_commit(&mma_bar);
  };
  const uint32_t lead = issuer ? elect_one() : 0u;
  // partial Gram matrices: [matrix][rank][iteration parity][128 x 128] fp32 in global memory (L2)
  float* sc_mat = scratch + (size_t)blockIdx.y * nc * 2 * RB * HD;

  for (int it = 0; it < iters; ++it) {
    const bool last = it == iters - 1;
    // ---------------- A = X^T X: partial over this rank's rows, summed over the cluster ----------------
    if (lead) {
#pragma unroll
      for (int ks = 0; ks < RB / 16; ++ks) {               // +2048 B per 16-row K step
        umma_ss(tb + C_A, d_xh_mn + 128 * ks, d_xh_mn + 128 * ks, idesc_mn, ks > 0);
        umma_ss(tb + C_A, d_xh_mn + 128 * ks, d_xl_mn + 128 * ks, idesc_mn, 1);
        umma_ss(tb + C_A, d_xl_mn + 128 * ks, d_xh_mn + 128 * ks, idesc_mn, 1);
      }
      tc_commit(&mma_bar);
    }
    __syncwarp();
    if (!issuer) {
      wait_mma();
      float v[32];
      {
        uint32_t r[32];
        tmem_ld_x32(tb + lane_base + C_A + 32 * cs, r);
        tc_wait_ld();
#pragma unroll
        for (int j = 0; j < 32; ++j) v[j] = __uint_as_float(r[j]);
      }
      rows_to_ex(v);
      worker_bar();
      float4* dst = reinterpret_cast<float4*>(sc_mat + ((size_t)rank * 2 + (it & 1)) * RB * HD);
#pragma unroll
      for (int k = 0; k < 8; ++k) dst[tid + THREADS * k] = *reinterpret_cast<const float4*>(ex_co(k));
    }
    cluster_arrive();                  // release at cluster scope: orders this rank's global writes for its peers
    cluster_wait();
    if (!issuer) {
      float4 a[8];
#pragma unroll
      for (int k = 0; k < 8; ++k) a[k] = make_float4(0.f, 0.f, 0.f, 0.f);
      for (uint32_t r = 0; r < nc; r += 2) {               // rank order: identical A on every rank
        const float4* s0 = reinterpret_cast<const float4*>(sc_mat + ((size_t)r * 2 + (it & 1)) * RB * HD);
        const float4* s1 = reinterpret_cast<const float4*>(sc_mat + ((size_t)(r + 1) * 2 + (it & 1)) * RB * HD);
        const bool two = r + 1 < nc;
        float4 p[8], p2[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          p[k] = __ldcg(s0 + tid + THREADS * k);
          p2[k] = two ? __ldcg(s1 + tid + THREADS * k) : make_float4(0.f, 0.f, 0.f, 0.f);
        }
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          a[k].x = (a[k].x + p[k].x) + p2[k].x; a[k].y = (a[k].y + p[k].y) + p2[k].y;
          a[k].z = (a[k].z + p[k].z) + p2[k].z; a[k].w = (a[k].w + p[k].w) + p2[k].w;
        }
      }
#pragma unroll
      for (int k = 0; k < 8; ++k) *reinterpret_cast<float4*>(ex_co(k)) = a[k];
      worker_bar();
      ex_to_rows(Areg);
      split_row32(Areg, AH, AL, trow, cs);
    }
    end_phase();
    // ---------------- Pm = a I + b A + c A A (A symmetric: K-major A . A^T) ----------------
    if (lead) product_k(tb + C_A2, d_ah, d_al, d_ah, d_al);
    __syncwarp();
    if (!issuer) {
      wait_mma();
      uint32_t r[32];
      tmem_ld_x32(tb + lane_base + C_A2 + 32 * cs, r);
      tc_wait_ld();
      float pm[32];
#pragma unroll
      for (int j = 0; j < 32; ++j) {
        float p = fmaf(cc, __uint_as_float(r[j]), cb * Areg[j]);
        if (32 * cs + j == trow) p += ca;
        pm[j] = p;
      }
      split_row32(pm, AH, AL, trow, cs);                   // the A tiles are dead: Pm takes their place
    }
    end_phase();
    // ---------------- X <- X Pm (Pm symmetric: K-major X . Pm^T) ----------------
    if (lead) product_k(tb + C_X, d_xh, d_xl, d_ah, d_al);
    __syncwarp();
    if (!issuer) {
      wait_mma();
      float x[32];
      {
        uint32_t r[32];
        tmem_ld_x32(tb + lane_base + C_X + 32 * cs, r);
        tc_wait_ld();
#pragma unroll
        for (int j = 0; j < 32; ++j) x[j] = __uint_as_float(r[j]);
      }
      if (!last) {
        split_row32(x, XH, XL, trow, cs);
      } else {
        asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
        // coalesced write-out through the staging tile: fused commit W <- W - NS(g) (Eq. 8), or NS(g) -> G
        rows_to_ex(x);
        worker_bar();
        if (Wm != nullptr) {
          float4* wm = reinterpret_cast<float4*>(Wm + blk);
          uint2* wb = reinterpret_cast<uint2*>(Wb + blk);
          uint2* wq = reinterpret_cast<uint2*>(Wq + blk);      // bf16 copy for the apply kernel
          float4 w[8];
#pragma unroll
          for (int k = 0; k < 8; ++k) w[k] = wm[tid + THREADS * k];
#pragma unroll
          for (int k = 0; k < 8; ++k) {
            const float4 d = *reinterpret_cast<const float4*>(ex_co(k));
            w[k].x -= d.x; w[k].y -= d.y; w[k].z -= d.z; w[k].w -= d.w;
            wm[tid + THREADS * k] = w[k];
            wb[tid + THREADS * k] = make_uint2(ttt_pack_wop2(w[k].x, w[k].y), ttt_pack_wop2(w[k].z, w[k].w));
            wq[tid + THREADS * k] = make_uint2(pack_bf16x2(w[k].x, w[k].y), pack_bf16x2(w[k].z, w[k].w));
          }
        } else {
          float4* gd = reinterpret_cast<float4*>(G + blk);
#pragma unroll
          for (int k = 0; k < 8; ++k) gd[tid + THREADS * k] = *reinterpret_cast<const float4*>(ex_co(k));
        }
      }
    }
    end_phase();
  }
  cluster_arrive();                    // no rank may exit while another still reads its s_part
  cluster_wait();
  if (warp == 0) tmem_dealloc(tb, 512);
}

int ns_tc_wide_supported(const ttt_config* cfg) {
  return cfg->act_dtype == TTT_BF16 && cfg->hd == nsw::HD && cfg->hidden % nsw::RB == 0 &&
         cfg->hidden >= 128 && cfg->hidden <= 1024 && !cfg->linear_fast_weight;
}

int launch_ns_tc_wide(ttt_ctx* ctx, bool fuse_commit, cudaStream_t s) {
  const ttt_config& c = ctx->cfg;
  if (!(ctx->attr_done & ATTR_NSW)) {
    TTT_CUDA_TRY(ctx, cudaFuncSetAttribute(ns_tc_wide_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                           (int)nsw::SMEM_BYTES), "ns_tc_wide_kernel smem attr");
    ctx->attr_done |= ATTR_NSW;
  }
  const int nc = c.hidden / nsw::RB;                       // cluster size: one CTA per 128-row block
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(nc, 3 * c.nh);
  cfg.blockDim = dim3(nsw::LAUNCH_THREADS);
  cfg.dynamicSmemBytes = nsw::SMEM_BYTES;
  cfg.stream = s;
  cudaLaunchAttribute attr[2];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = nc;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[1].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 2;
  float* G = ctx->G;
  const float* P = ctx->partials;
  int n_sets = ctx->n_partials, use_G = ctx->G_valid ? 1 : 0, H = c.hidden, iters = c.ns_iters;
  size_t set_elems = 3 * ctx->mat_elems;
  float* Wm = fuse_commit ? ctx->Wm : nullptr;
  ttt_wop_t* Wb = fuse_commit ? ctx->Wb : nullptr;
  cudaError_t e = cudaLaunchKernelEx(&cfg, ns_tc_wide_kernel, G, P, n_sets, set_elems, use_G, H, iters, Wm, Wb, ctx->Wq, ctx->ns_scratch);
  if (e != cudaSuccess) return set_error(ctx, TTT_ERR_CUDA, "ns_tc_wide_kernel launch", e);
  TTT_LAUNCH_CHECK(ctx, "ns_tc_wide_kernel");
  ctx->G_valid = !fuse_commit;
  ctx->n_partials = 0;
  return TTT_OK;
}

}  // namespace ttt
