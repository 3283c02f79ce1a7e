// streamkl_bwd_sm100.cuh -- StreamKL backward by recomputation for sm_100a.
//
// One kernel template, two instantiations per problem ("separate dQ / dK kernels", both
// deterministic and atomic-free because every output tile has exactly one owner):
//   OWNER_K = false : CTA owns a 128-row Q tile, streams 64-key tiles      -> dQ1, dQ2   (Alg.2 :224-234, Alg.3 :255-286)
//   OWNER_K = true  : CTA owns a 128-row K tile, streams 64-query tiles    -> dK1, dK2   (transposed tiling, :294, :309)
// With X the owner side and Y the streamed side, per step:
//   S1' = X1 Y1^T, S2' = X2 Y2^T        tcgen05.mma -> TMEM (lane = owner row)                                   (B2)
//   P_t = exp2(S_t' sc_t - lse_t log2e)  recomputed from the saved LSE (:216)                                     (B3)
//   dS2 = g (P2 - P1)   [fp32 subtract, one bf16 rounding]      dS1 = g P1 ((s1 - s2) - (lse1 - lse2) - kl)  Eq.12 (B4)
//   dX2 += dS2 Y2,  dX1 += dS1 Y1       tcgen05.mma, A = dS from swizzled smem, B = the Y tile read MN-major,
//                                        accumulators stay in TMEM for the whole CTA                               (B5)
// Epilogue: dX * c_t -> bf16 -> HBM, one rounding (B6).
// Warp roles: warp 0 TMA producer (+ per-query scalars when OWNER_K), warp 1 MMA issuer, warp 2 TMEM allocator,
// warps 4-7 / 8-11 two softmax warpgroups that take alternate steps (each has its own S' stage and dS buffer).
#pragma once
#include <cuda_bf16.h>
#include <math_constants.h>

#include "sm100_ptx.cuh"

namespace skl {

template <int D1, int D2, bool TEACHER>
struct BwdCfg {
  static_assert(D1 % 64 == 0 && D2 % 64 == 0 && D1 <= 128 && D2 <= 128, "tcgen05 path: d in {64,128}");
  static constexpr int BX = 128;   // owner rows per CTA (TMEM lanes)
  static constexpr int BY = 64;    // streamed rows per step
  static constexpr int KB1 = D1 / 64, KB2 = D2 / 64;
  static constexpr int XBLK = BX * 128, YBLK = BY * 128;
  static constexpr int X_BYTES = (KB1 + KB2) * XBLK;
  static constexpr int DS_TILE = BX * BY * 2;                        // one [128 x 64] bf16 dS tile
  static constexpr int DS_PER_WG = (TEACHER ? 2 : 1) * DS_TILE;
  static constexpr int DS_BYTES = 2 * DS_PER_WG;
  static constexpr int Y_STAGE = (KB1 + KB2) * YBLK;
  static constexpr int STAT_STAGE = BY * 16;                         // float4 per streamed query (OWNER_K)
  static constexpr int AUX_BYTES = 512;
  static constexpr int NSTAGE_RAW = (227 * 1024 - 1024 - AUX_BYTES - X_BYTES - DS_BYTES) / (Y_STAGE + STAT_STAGE);
  static constexpr int NSTAGE = NSTAGE_RAW > 6 ? 6 : NSTAGE_RAW;
  static_assert(NSTAGE >= 2, "need at least a double-buffered Y ring");
  static constexpr int SMEM_BYTES = 1024 + X_BYTES + DS_BYTES + NSTAGE * (Y_STAGE + STAT_STAGE) + AUX_BYTES;
  static constexpr int THREADS = 384;
  static constexpr uint32_t TMEM_COLS = 512;
  static constexpr uint32_t COL_DX1 = 256, COL_DX2 = 256 + (TEACHER ? D1 : 0);   // after the two S' stages (2 x 128)
};

struct BwdParams {
  int NQ, NK, TX, BH;
  float c1, c2;
  const float* kl;
  const float* lse1;
  const float* lse2;
  const float* dkl;
  __nv_bfloat16* dX1;   // dQ1 or dK1 (nullptr when !TEACHER)
  __nv_bfloat16* dX2;   // dQ2 or dK2
};

__device__ __forceinline__ uint32_t pack_bf16x2(float lo, float hi) {
  uint32_t r;
  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
  return r;
}

// dX accumulator (this warp's 32 lanes x NCOLS fp32 columns) -> * scale -> bf16 -> global row
template <int NCOLS>
__device__ __forceinline__ void store_dx_row(uint32_t taddr, float scale, __nv_bfloat16* out_row, bool valid) {
#pragma unroll
  for (int c0 = 0; c0 < NCOLS; c0 += 32) {
    uint32_t v[32];
    tmem_ld32(taddr + c0, v);
    tmem_wait_ld();
    if (valid) {
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        uint4 o;
        o.x = pack_bf16x2(__uint_as_float(v[q * 8 + 0]) * scale, __uint_as_float(v[q * 8 + 1]) * scale);
        o.y = pack_bf16x2(__uint_as_float(v[q * 8 + 2]) * scale, __uint_as_float(v[q * 8 + 3]) * scale);
        o.z = pack_bf16x2(__uint_as_float(v[q * 8 + 4]) * scale, __uint_as_float(v[q * 8 + 5]) * scale);
        o.w = pack_bf16x2(__uint_as_float(v[q * 8 + 6]) * scale, __uint_as_float(v[q * 8 + 7]) * scale);
        *reinterpret_cast<uint4*>(out_row + c0 + q * 8) = o;
      }
    }
  }
}

template <int D1, int D2, bool CAUSAL, bool TEACHER, bool OWNER_K>
__global__ void __launch_bounds__(384, 1)
streamkl_bwd_sm100_kernel(const __grid_constant__ CUtensorMap tmQ1, const __grid_constant__ CUtensorMap tmK1,
                          const __grid_constant__ CUtensorMap tmQ2, const __grid_constant__ CUtensorMap tmK2, const BwdParams p) {
  using C = BwdCfg<D1, D2, TEACHER>;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t* sX1 = smem;
  uint8_t* sX2 = sX1 + C::KB1 * C::XBLK;
  uint8_t* sDS = smem + C::X_BYTES;                       // [wg][{dS2, dS1}] 16 KB tiles
  uint8_t* sY = sDS + C::DS_BYTES;                        // NSTAGE x {Y1 blocks, Y2 blocks}
  float4* sStat = reinterpret_cast<float4*>(sY + C::NSTAGE * C::Y_STAGE);   // NSTAGE x BY float4
  uint64_t* bars = reinterpret_cast<uint64_t*>(reinterpret_cast<uint8_t*>(sStat) + C::NSTAGE * C::STAT_STAGE);
  uint64_t* x_full = bars;                       // 1
  uint64_t* y_full = bars + 1;                   // NSTAGE
  uint64_t* y_empty = y_full + C::NSTAGE;        // NSTAGE
  uint64_t* s_full = y_empty + C::NSTAGE;        // 2 (per softmax WG)
  uint64_t* s_empty = s_full + 2;                // 2
  uint64_t* ds_full = s_empty + 2;               // 2
  uint64_t* ds_empty = ds_full + 2;              // 2
  uint64_t* dx_full = ds_empty + 2;              // 1
  uint32_t* tmem_ptr = reinterpret_cast<uint32_t*>(dx_full + 1);

  const CUtensorMap* tmX1 = OWNER_K ? &tmK1 : &tmQ1;
  const CUtensorMap* tmX2 = OWNER_K ? &tmK2 : &tmQ2;
  const CUtensorMap* tmY1 = OWNER_K ? &tmQ1 : &tmK1;
  const CUtensorMap* tmY2 = OWNER_K ? &tmQ2 : &tmK2;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int bh = blockIdx.x / p.TX;
  // heavy tiles first: late Q tiles see more keys, early K tiles are seen by more queries
  const int xt = (CAUSAL && !OWNER_K) ? (p.TX - 1 - (blockIdx.x % p.TX)) : (blockIdx.x % p.TX);
  const int x0 = xt * C::BX;
  const int off = p.NK - p.NQ;
  const int NX = OWNER_K ? p.NK : p.NQ;
  const int NY = OWNER_K ? p.NQ : p.NK;
  int j_begin = 0, j_end = (NY + C::BY - 1) / C::BY;
  if (CAUSAL) {
    if (OWNER_K) j_begin = max(0, x0 - off) / C::BY;                       // first query that sees key x0
    else         j_end = min(p.NK - 1, x0 + C::BX - 1 + off) / C::BY + 1;   // last key the tile's last row sees
  }
  const int nsteps = max(0, j_end - j_begin);

  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tmQ1); tma_prefetch_desc(&tmK1); tma_prefetch_desc(&tmQ2); tma_prefetch_desc(&tmK2);
  }
  if (warp == 1 && lane == 0) {
    mbar_init(x_full, 1);
    for (int s = 0; s < C::NSTAGE; ++s) { mbar_init(&y_full[s], 1); mbar_init(&y_empty[s], 1); }
    for (int w = 0; w < 2; ++w) {
      mbar_init(&s_full[w], 1); mbar_init(&s_empty[w], 4);
      mbar_init(&ds_full[w], 4); mbar_init(&ds_empty[w], 1);
    }
    mbar_init(dx_full, 1);
    fence_mbar_init();
  }
  if (warp == 2) tmem_alloc<C::TMEM_COLS>(tmem_ptr);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_ptr;
  const float L2E = 1.4426950408889634f;

  if (warp == 0) {
    // ===================== producer =====================
    uint64_t pol_x = 0, pol_y = 0;
    if (lane == 0) {
      pol_x = l2_policy_evict_first(); pol_y = l2_policy_evict_last();
      mbar_arrive_expect_tx(x_full, C::X_BYTES);
#pragma unroll
      for (int kb = 0; kb < C::KB1; ++kb) tma_load_3d_hint(sX1 + kb * C::XBLK, tmX1, x_full, kb * 64, x0, bh, pol_x);
#pragma unroll
      for (int kb = 0; kb < C::KB2; ++kb) tma_load_3d_hint(sX2 + kb * C::XBLK, tmX2, x_full, kb * 64, x0, bh, pol_x);
    }
    for (int it = 0; it < nsteps; ++it) {
      const int j = j_begin + it;
      const int s = it % C::NSTAGE;
      const uint32_t ph = (it / C::NSTAGE) & 1;
      if (lane == 0) mbar_wait(&y_empty[s], ph ^ 1);
      __syncwarp();
      if (OWNER_K) {  // per-query scalars of the streamed query tile -> shared (B1)
#pragma unroll
        for (int t = 0; t < C::BY / 32; ++t) {
          const int qi = j * C::BY + t * 32 + lane;
          float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
          if (qi < p.NQ) {
            const size_t o = size_t(bh) * p.NQ + qi;
            const float a = p.lse1[o], b = p.lse2[o];
            v = make_float4(a * L2E, b * L2E, p.dkl[o], (a - b) + p.kl[o]);
          }
          sStat[s * C::BY + t * 32 + lane] = v;
        }
        __syncwarp();
      }
      if (lane == 0) {
        mbar_arrive_expect_tx(&y_full[s], C::Y_STAGE);
        uint8_t* st = sY + s * C::Y_STAGE;
#pragma unroll
        for (int kb = 0; kb < C::KB1; ++kb) tma_load_3d_hint(st + kb * C::YBLK, tmY1, &y_full[s], kb * 64, j * C::BY, bh, pol_y);
#pragma unroll
        for (int kb = 0; kb < C::KB2; ++kb)
          tma_load_3d_hint(st + (C::KB1 + kb) * C::YBLK, tmY2, &y_full[s], kb * 64, j * C::BY, bh, pol_y);
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer =====================
    if (lane == 0 && nsteps > 0) {
      constexpr uint32_t idesc_s = umma_idesc_bf16(C::BX, C::BY, 0, 0);      // S' = X Y^T   : A,B K-major
      constexpr uint32_t idesc_g1 = umma_idesc_bf16(C::BX, D1, 0, 1);        // dX1 += dS1 Y1: B MN-major
      constexpr uint32_t idesc_g2 = umma_idesc_bf16(C::BX, D2, 0, 1);
      const uint32_t x1addr = smem_u32(sX1), x2addr = smem_u32(sX2);
      mbar_wait(x_full, 0);
      tc_fence_after();
      auto issue_S = [&](int it) {
        const int s = it % C::NSTAGE;
        const uint32_t ph = (it / C::NSTAGE) & 1;
        const int w = it & 1;
        const uint32_t wph = (it >> 1) & 1;
        mbar_wait(&y_full[s], ph);
        mbar_wait(&s_empty[w], wph ^ 1);
        tc_fence_after();
        const uint32_t yaddr = smem_u32(sY + s * C::Y_STAGE);
        const uint32_t dS1 = tmem_base + w * 128, dS2 = dS1 + 64;
#pragma unroll
        for (int kb = 0; kb < C::KB1; ++kb)
#pragma unroll
          for (int k = 0; k < 4; ++k)
            umma_bf16_ss(dS1, umma_smem_desc_sw128(x1addr + kb * C::XBLK + k * 32, 16, 1024),
                         umma_smem_desc_sw128(yaddr + kb * C::YBLK + k * 32, 16, 1024), idesc_s, (kb | k) != 0);
#pragma unroll
        for (int kb = 0; kb < C::KB2; ++kb)
#pragma unroll
          for (int k = 0; k < 4; ++k)
            umma_bf16_ss(dS2, umma_smem_desc_sw128(x2addr + kb * C::XBLK + k * 32, 16, 1024),
                         umma_smem_desc_sw128(yaddr + (C::KB1 + kb) * C::YBLK + k * 32, 16, 1024), idesc_s, (kb | k) != 0);
        umma_commit(&s_full[w]);
      };
      auto issue_dX = [&](int it) {
        const int s = it % C::NSTAGE;
        const int w = it & 1;
        const uint32_t wph = (it >> 1) & 1;
        mbar_wait(&ds_full[w], wph);
        tc_fence_after();
        const uint32_t yaddr = smem_u32(sY + s * C::Y_STAGE);
        const uint32_t dsaddr = smem_u32(sDS + w * C::DS_PER_WG);
        const uint32_t acc = it > 0;
        // dX2 += dS2 (128 x 64, K-major) * Y2 (64 x D2 read MN-major: 64-column chunks YBLK apart, 8-row groups 1024 B apart)
#pragma unroll
        for (int k = 0; k < 4; ++k)
          umma_bf16_ss(tmem_base + C::COL_DX2, umma_smem_desc_sw128(dsaddr + k * 32, 16, 1024),
                       umma_smem_desc_sw128(yaddr + C::KB1 * C::YBLK + k * 2048, C::YBLK, 1024), idesc_g2, acc | (k != 0));
        if (TEACHER) {
#pragma unroll
          for (int k = 0; k < 4; ++k)
            umma_bf16_ss(tmem_base + C::COL_DX1, umma_smem_desc_sw128(dsaddr + C::DS_TILE + k * 32, 16, 1024),
                         umma_smem_desc_sw128(yaddr + k * 2048, C::YBLK, 1024), idesc_g1, acc | (k != 0));
        }
        umma_commit(&ds_empty[w]);
        umma_commit(&y_empty[s]);
      };
      issue_S(0);
      for (int it = 0; it < nsteps; ++it) {
        if (it + 1 < nsteps) issue_S(it + 1);   // keep the tensor pipe busy while the softmax warps work on step `it`
        issue_dX(it);
      }
      umma_commit(dx_full);
    }
  } else if (warp >= 4) {
    // ===================== softmax / dS warpgroups =====================
    const int w = (warp - 4) >> 2;
    const int quarter = warp & 3;
    const int rloc = quarter * 32 + lane;     // owner row within the tile = TMEM lane
    const int xrow = x0 + rloc;
    const float sc1 = p.c1 * L2E, sc2 = p.c2 * L2E;
    float my_L1 = 0.f, my_L2 = 0.f, my_g = 0.f, my_term = 0.f;
    if (!OWNER_K && xrow < p.NQ) {
      const size_t o = size_t(bh) * p.NQ + xrow;
      const float a = p.lse1[o], b = p.lse2[o];
      my_L1 = a * L2E; my_L2 = b * L2E; my_g = p.dkl[o]; my_term = (a - b) + p.kl[o];
    }
    uint8_t* ds2_row = sDS + w * C::DS_PER_WG + rloc * 128;
    uint8_t* ds1_row = ds2_row + C::DS_TILE;
    const int sw = rloc & 7;
    for (int it = w; it < nsteps; it += 2) {
      const int j = j_begin + it;
      const int s = it % C::NSTAGE;
      const uint32_t wph = (it >> 1) & 1;
      mbar_wait(&s_full[w], wph);
      tc_fence_after();
      const uint32_t taddr = tmem_base + (uint32_t(quarter * 32) << 16) + w * 128;
      uint32_t r1[64], r2[64];
      tmem_ld32(taddr, *reinterpret_cast<uint32_t(*)[32]>(&r1[0]));
      tmem_ld32(taddr + 32, *reinterpret_cast<uint32_t(*)[32]>(&r1[32]));
      tmem_ld32(taddr + 64, *reinterpret_cast<uint32_t(*)[32]>(&r2[0]));
      tmem_ld32(taddr + 96, *reinterpret_cast<uint32_t(*)[32]>(&r2[32]));
      tmem_wait_ld();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&s_empty[w]);
      const int ybase = j * C::BY;
      // tile-uniform: does any (query,key) pair of this tile fall outside the causal mask?
      // (a streamed KEY tail is masked too: TMA zero-fills those rows, but P = exp2(0 - lse) may overflow and inf * 0 = NaN)
      const bool masked = (CAUSAL && (OWNER_K ? (ybase + off < x0 + C::BX - 1) : (ybase + C::BY - 1 > x0 + off))) ||
                          (!OWNER_K && ybase + C::BY > p.NK);
      mbar_wait(&ds_empty[w], wph ^ 1);   // the dX MMAs of this warpgroup's previous step have consumed the dS buffer
      const float4* stat = sStat + s * C::BY;
#pragma unroll
      for (int c = 0; c < 8; ++c) {
        uint32_t o2[4], o1[4];
#pragma unroll
        for (int h = 0; h < 4; ++h) {
          float d2v[2], d1v[2];
#pragma unroll
          for (int u = 0; u < 2; ++u) {
            const int e = c * 8 + h * 2 + u;
            float L1 = my_L1, L2 = my_L2, g = my_g, term = my_term;
            if (OWNER_K) { const float4 t = stat[e]; L1 = t.x; L2 = t.y; g = t.z; term = t.w; }
            const float s1 = __uint_as_float(r1[e]), s2 = __uint_as_float(r2[e]);
            const float p1 = ex2_approx(fmaf(s1, sc1, -L1));      // P1 = exp(s1 - lse1)   (Alg.2 line 7)
            const float p2 = ex2_approx(fmaf(s2, sc2, -L2));
            float a2 = g * (p2 - p1);                              // dS2 (Alg.2 line 8): fp32 subtract, rounded once below
            float a1 = 0.f;
            if (TEACHER) a1 = (g * p1) * (fmaf(s1, p.c1, -term) - s2 * p.c2);   // dS1 (Alg.3 lines 9-10, Eq.12)
            if (masked) {
              const bool ok = OWNER_K ? (xrow <= ybase + e + off) : ((ybase + e < p.NK) && (!CAUSAL || ybase + e <= xrow + off));
              a2 = ok ? a2 : 0.f;
              a1 = ok ? a1 : 0.f;
            }
            d2v[u] = a2; d1v[u] = a1;
          }
          o2[h] = pack_bf16x2(d2v[0], d2v[1]);
          if (TEACHER) o1[h] = pack_bf16x2(d1v[0], d1v[1]);
        }
        const int chunk = (c ^ sw) << 4;   // 128-byte swizzle: 16-byte chunk index XOR (row mod 8)
        *reinterpret_cast<uint4*>(ds2_row + chunk) = make_uint4(o2[0], o2[1], o2[2], o2[3]);
        if (TEACHER) *reinterpret_cast<uint4*>(ds1_row + chunk) = make_uint4(o1[0], o1[1], o1[2], o1[3]);
      }
      fence_proxy_async_smem();   // generic-proxy stores -> visible to the tensor core's async-proxy reads
      __syncwarp();
      if (lane == 0) mbar_arrive(&ds_full[w]);
    }
    // ---- epilogue: dX (TMEM fp32) * c_t -> bf16 -> HBM
    const bool valid = xrow < NX;
    const uint32_t lane_addr = tmem_base + (uint32_t(quarter * 32) << 16);
    const size_t orow = size_t(bh) * NX + (valid ? xrow : 0);
    if (nsteps > 0) {
      mbar_wait(dx_full, 0);
      tc_fence_after();
      if (TEACHER) {
        if (w == 0) store_dx_row<D1>(lane_addr + C::COL_DX1, p.c1, p.dX1 + orow * D1, valid);
        else        store_dx_row<D2>(lane_addr + C::COL_DX2, p.c2, p.dX2 + orow * D2, valid);
      } else {
        store_dx_row<D2 / 2>(lane_addr + C::COL_DX2 + w * (D2 / 2), p.c2, p.dX2 + orow * D2 + w * (D2 / 2), valid);
      }
    } else if (valid) {
      const uint4 z = make_uint4(0, 0, 0, 0);
      if (w == 0) { for (int c = 0; c < D2; c += 8) *reinterpret_cast<uint4*>(p.dX2 + orow * D2 + c) = z; }
      else if (TEACHER) { for (int c = 0; c < D1; c += 8) *reinterpret_cast<uint4*>(p.dX1 + orow * D1 + c) = z; }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 2) {
    tc_fence_after();
    tmem_dealloc<C::TMEM_COLS>(tmem_base);
  }
}

}  // namespace skl
