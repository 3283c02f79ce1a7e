// streamkl_bwd_wide_sm100.cuh -- the owner backward kernels (streamkl_bwd_sm100.cuh) for head dims above 128 (padded to
// 192 / 256; PAPER.md:216, :288: backward by recomputation; :313-315 separate dQ / dK kernels by tile ownership).
//
// What changes against the fixed-plan kernel is only where the operands live, because the budgets no longer close:
//   * TMEM: the dX accumulators need one fp32 column per head-dim element.  S' (128) + dS (128) leave 256 columns, so a
//     launch differentiates ONE distribution (GRAD = 1: dX1 only, the teacher pass; GRAD = 2: dX2 only, the student pass)
//     unless d1 + d2 <= 256 padded (GRAD = 3: both, as the fixed plans do).  Setting 2 with d1 + d2 > 256 is therefore two
//     passes per owner side; every pass recomputes both logit tiles (dS1 needs s1 - s2 and P1, dS2 needs P1 and P2).
//   * shared memory: the owner tile alone is up to 128 KB, so the streamed side is kept in TWO rings, one per distribution,
//     of whole [64 rows x d_t] stages.  A stage of a distribution that is not differentiated is released as soon as its
//     logit MMAs retire; a stage of a differentiated one stays until the dX MMAs that read it (as the MN-major B operand)
//     retire.  The numbers of 64-element K-blocks per row (kb1, kb2), the ring depths and the number of S' stages are
//     run-time kernel parameters: one instantiation per (CAUSAL, GRAD, OWNER_K) covers every wide head-dim pair.
// Warp roles, barriers' protocol, the dS arithmetic (ds_row) and the epilogue are those of streamkl_bwd_sm100.cuh.
#pragma once
#include "streamkl_bwd_sm100.cuh"

namespace skl {

struct BwdWideCfg {
  static constexpr int BX = 128, BY = 64;
  static constexpr int XBLK = BX * 128, YBLK = BY * 128;   // one [rows x 64 elements] swizzled block
  static constexpr int STAT_STAGE = BY * 16;
  static constexpr int MAX_STAGES = 4;
  static constexpr int AUX_BYTES = 512;
  static constexpr int SMEM_LIMIT = 227 * 1024;
  static constexpr int THREADS = 128 + 512;
  static constexpr uint32_t TMEM_COLS = 512;
};

struct BwdWideParams {
  BwdParams b;
  int kb1, kb2;   // 64-element K-blocks per row of distribution 1 / 2 (padded head dim / 64)
  int ns1, ns2;   // ring depth (stages of 64 streamed rows) per distribution
  int nss;        // S' stages in TMEM (2 if they fit beside dS and dX, else 1)
  uint32_t smem_need;   // bytes used from the 1024-byte-aligned base (the launch adds whatever alignment slack still fits)
};

// GRAD: bit 0 = differentiate distribution 1 (dX1: dQ1 / dK1), bit 1 = distribution 2 (dX2).
template <bool CAUSAL, int GRAD, bool OWNER_K>
__global__ void __launch_bounds__(BwdWideCfg::THREADS, 1)
streamkl_bwd_wide_sm100_kernel(const __grid_constant__ CUtensorMap tmQ1, const __grid_constant__ CUtensorMap tmK1,
                               const __grid_constant__ CUtensorMap tmQ2, const __grid_constant__ CUtensorMap tmK2,
                               const __grid_constant__ BwdWideParams pw) {
  using C = BwdWideCfg;
  static_assert(GRAD >= 1 && GRAD <= 3, "GRAD: 1 teacher pass, 2 student pass, 3 both");
  constexpr bool G1 = (GRAD & 1) != 0, G2 = (GRAD & 2) != 0;
  const BwdParams& p = pw.b;
  const int KB1 = pw.kb1, KB2 = pw.kb2, NS1 = pw.ns1, NS2 = pw.ns2, NSS = pw.nss;
  const int D1 = KB1 * 64, D2 = KB2 * 64;                       // padded head dims
  const int Y1_STAGE = KB1 * C::YBLK, Y2_STAGE = KB2 * C::YBLK;
  // the streamed queries' scalars (OWNER_K) ride with the ring of a differentiated distribution: that stage is released by
  // the dX MMAs, i.e. after the dS warps have read them
  constexpr bool STAT_ON_2 = G2;
  const int NST = STAT_ON_2 ? NS2 : NS1;

  extern __shared__ __align__(1024) uint8_t smem_wide[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_wide) + 1023) & ~uintptr_t(1023));
  {
    // the largest pairs (X 128 KB + three 32 KB stages) leave less than 1 KB of slack: the dynamic window is 1024-byte aligned in
    // practice (then nothing is lost to the round-up above); if it ever is not, fail loudly instead of overrunning it
    uint32_t dyn;
    asm volatile("mov.u32 %0, %%dynamic_smem_size;" : "=r"(dyn));
    if (uint32_t(smem - smem_wide) + pw.smem_need > dyn) __trap();
  }
  uint8_t* sX1 = smem;
  uint8_t* sX2 = sX1 + KB1 * C::XBLK;
  uint8_t* sY1 = sX2 + KB2 * C::XBLK;
  uint8_t* sY2 = sY1 + NS1 * Y1_STAGE;
  float4* sStat = reinterpret_cast<float4*>(sY2 + NS2 * Y2_STAGE);
  uint64_t* bars = reinterpret_cast<uint64_t*>(reinterpret_cast<uint8_t*>(sStat) + (OWNER_K ? NST * C::STAT_STAGE : 0));
  uint64_t* x_full = bars;                          // 1
  uint64_t* y1_full = bars + 1;                     // MAX_STAGES
  uint64_t* y1_empty = y1_full + C::MAX_STAGES;
  uint64_t* y2_full = y1_empty + C::MAX_STAGES;
  uint64_t* y2_empty = y2_full + C::MAX_STAGES;
  uint64_t* s_full = y2_empty + C::MAX_STAGES;      // 2 (per parity group)
  uint64_t* s_empty = s_full + 2;
  uint64_t* ds_full = s_empty + 2;
  uint64_t* ds_empty = ds_full + 2;
  uint64_t* dx_full = ds_empty + 2;                 // 1
  uint32_t* tmem_ptr = reinterpret_cast<uint32_t*>(dx_full + 1);

  const CUtensorMap* tmX1 = OWNER_K ? &tmK1 : &tmQ1;
  const CUtensorMap* tmX2 = OWNER_K ? &tmK2 : &tmQ2;
  const CUtensorMap* tmY1 = OWNER_K ? &tmQ1 : &tmK1;
  const CUtensorMap* tmY2 = OWNER_K ? &tmQ2 : &tmK2;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int unit = blockIdx.x / p.TX;
  const int HX = OWNER_K ? p.HK : p.H;
  const int bx = unit / HX, hx = unit % HX;
  const int xt = (CAUSAL && !OWNER_K) ? (p.TX - 1 - (blockIdx.x % p.TX)) : (blockIdx.x % p.TX);
  const int x0 = xt * C::BX;
  const int off = p.NK - p.NQ;
  const int NX = OWNER_K ? p.NK : p.NQ;
  const int NY = OWNER_K ? p.NQ : p.NK;
  const long long NQP = bwd_stats_padded_rows(p.NQ);
  int j_begin = 0, j_end = (NY + C::BY - 1) / C::BY;
  if (CAUSAL) {
    if (OWNER_K) j_begin = max(0, x0 - off) / C::BY;
    else         j_end = min(p.NK - 1, x0 + C::BX - 1 + off) / C::BY + 1;
  }
  const int nsteps1 = max(0, j_end - j_begin);
  const int nsteps = nsteps1 * (OWNER_K ? p.G : 1);
  auto step_g = [&](int it) { return OWNER_K ? it / max(nsteps1, 1) : 0; };
  auto step_j = [&](int it) { return j_begin + (OWNER_K ? it % max(nsteps1, 1) : it); };

  // TMEM columns: NSS x {S1' 64, S2' 64} | 2 x {dS1 32, dS2 32} | dX1 (D1 if G1) | dX2 (D2 if G2)
  const uint32_t COL_DS = NSS * 128, COL_DX1 = COL_DS + 128, COL_DX2 = COL_DX1 + (G1 ? D1 : 0);

  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tmQ1); tma_prefetch_desc(&tmK1); tma_prefetch_desc(&tmQ2); tma_prefetch_desc(&tmK2);
  }
  if (warp == 1 && lane == 0) {
    mbar_init(x_full, 1);
    for (int s = 0; s < C::MAX_STAGES; ++s) {
      mbar_init(&y1_full[s], 1); mbar_init(&y1_empty[s], 1);
      mbar_init(&y2_full[s], 1); mbar_init(&y2_empty[s], 1);
    }
    for (int w = 0; w < 2; ++w) {
      mbar_init(&s_full[w], 1); mbar_init(&s_empty[w], 8);
      mbar_init(&ds_full[w], 8); mbar_init(&ds_empty[w], 1);
    }
    mbar_init(dx_full, 1);
    fence_mbar_init();
  }
  if (warp == 2) tmem_alloc<C::TMEM_COLS>(tmem_ptr);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_ptr;

  if (warp < 4) {
    reg_dealloc<32>();
    if (warp == 0) {
      // ===================== producer =====================
      if (lane == 0) {
        const uint64_t pol_x = l2_policy_evict_first(), pol_y = l2_policy_evict_last();
        mbar_arrive_expect_tx(x_full, uint32_t((KB1 + KB2) * C::XBLK));
        for (int kb = 0; kb < KB1; ++kb) tma_load_4d_hint(sX1 + kb * C::XBLK, tmX1, x_full, kb * 64, x0, hx, bx, pol_x);
        for (int kb = 0; kb < KB2; ++kb) tma_load_4d_hint(sX2 + kb * C::XBLK, tmX2, x_full, kb * 64, x0, hx, bx, pol_x);
        int s1 = 0, s2 = 0;
        uint32_t ph1 = 0, ph2 = 0;
        for (int it = 0; it < nsteps; ++it) {
          const int j = step_j(it);
          const int hy = OWNER_K ? hx * p.G + step_g(it) : hx / p.G;
          const void* stat_src = p.stats + (size_t(bx * p.H + hy) * NQP + size_t(j) * C::BY);
          mbar_wait(&y1_empty[s1], ph1 ^ 1);
          mbar_arrive_expect_tx(&y1_full[s1], uint32_t(Y1_STAGE + ((OWNER_K && !STAT_ON_2) ? C::STAT_STAGE : 0)));
          for (int kb = 0; kb < KB1; ++kb)
            tma_load_4d_hint(sY1 + s1 * Y1_STAGE + kb * C::YBLK, tmY1, &y1_full[s1], kb * 64, j * C::BY, hy, bx, pol_y);
          if (OWNER_K && !STAT_ON_2) bulk_load_1d(sStat + s1 * C::BY, stat_src, C::STAT_STAGE, &y1_full[s1]);
          mbar_wait(&y2_empty[s2], ph2 ^ 1);
          mbar_arrive_expect_tx(&y2_full[s2], uint32_t(Y2_STAGE + ((OWNER_K && STAT_ON_2) ? C::STAT_STAGE : 0)));
          for (int kb = 0; kb < KB2; ++kb)
            tma_load_4d_hint(sY2 + s2 * Y2_STAGE + kb * C::YBLK, tmY2, &y2_full[s2], kb * 64, j * C::BY, hy, bx, pol_y);
          if (OWNER_K && STAT_ON_2) bulk_load_1d(sStat + s2 * C::BY, stat_src, C::STAT_STAGE, &y2_full[s2]);
          if (++s1 == NS1) { s1 = 0; ph1 ^= 1; }
          if (++s2 == NS2) { s2 = 0; ph2 ^= 1; }
        }
      }
    } else if (warp == 1) {
      // ===================== S' MMA issuer =====================
      const uint32_t idesc_s = umma_idesc_16(C::BX, C::BY, 0, 0, p.fmt16);
      const uint64_t dx1 = umma_smem_desc_sw128(smem_u32(sX1), 16, 1024);
      const uint64_t dx2 = umma_smem_desc_sw128(smem_u32(sX2), 16, 1024);
      const uint64_t dy1 = umma_smem_desc_sw128(smem_u32(sY1), 16, 1024);
      const uint64_t dy2 = umma_smem_desc_sw128(smem_u32(sY2), 16, 1024);
      if (nsteps > 0) {
        mbar_wait(x_full, 0);
        tc_fence_after();
      }
      int s1 = 0, s2 = 0, ss = 0;
      uint32_t ph1 = 0, ph2 = 0;
      for (int it = 0; it < nsteps; ++it) {
        const int prev = it - NSS;                    // the step whose logits this S' stage held last
        if (prev >= 0) mbar_wait(&s_empty[prev & 1], (prev >> 1) & 1);
        const uint32_t tS1 = tmem_base + ss * 128, tS2 = tS1 + 64;
        mbar_wait(&y1_full[s1], ph1);
        tc_fence_after();
        {
          const uint64_t a = dx1, b = dy1 + uint64_t((s1 * Y1_STAGE) >> 4);
          if (elect_one()) {
            for (int kb = 0; kb < KB1; ++kb)
#pragma unroll
              for (int k = 0; k < 4; ++k)
                umma_bf16_ss(tS1, a + uint64_t((kb * C::XBLK + k * 32) >> 4), b + uint64_t((kb * C::YBLK + k * 32) >> 4), idesc_s, (kb | k) != 0);
            if (!G1) umma_commit(&y1_empty[s1]);        // not differentiated: the stage is free once its logits exist
          }
          __syncwarp();
        }
        mbar_wait(&y2_full[s2], ph2);
        tc_fence_after();
        {
          const uint64_t a = dx2, b = dy2 + uint64_t((s2 * Y2_STAGE) >> 4);
          if (elect_one()) {
            for (int kb = 0; kb < KB2; ++kb)
#pragma unroll
              for (int k = 0; k < 4; ++k)
                umma_bf16_ss(tS2, a + uint64_t((kb * C::XBLK + k * 32) >> 4), b + uint64_t((kb * C::YBLK + k * 32) >> 4), idesc_s, (kb | k) != 0);
            if (!G2) umma_commit(&y2_empty[s2]);
            umma_commit(&s_full[it & 1]);
          }
          __syncwarp();
        }
        if (++s1 == NS1) { s1 = 0; ph1 ^= 1; }
        if (++s2 == NS2) { s2 = 0; ph2 ^= 1; }
        if (++ss == NSS) ss = 0;
      }
    } else if (warp == 3) {
      // ===================== dX MMA issuer =====================
      const uint32_t idesc_g1 = umma_idesc_16(C::BX, D1, 0, 1, p.fmt16);       // dX1 += dS1 Y1: A from TMEM, B MN-major, N = d1 (<= 256)
      const uint32_t idesc_g2 = umma_idesc_16(C::BX, D2, 0, 1, p.fmt16);
      // Y as the MN-major B operand: 64-column chunks YBLK apart (LBO), 8-row groups 1024 B apart (SBO); a K=16 slice = 2048 B
      const uint64_t dm1 = umma_smem_desc_sw128(smem_u32(sY1), C::YBLK, 1024);
      const uint64_t dm2 = umma_smem_desc_sw128(smem_u32(sY2), C::YBLK, 1024);
      int s1 = 0, s2 = 0;
      for (int it = 0; it < nsteps; ++it) {
        const int st = it & 1;
        mbar_wait(&ds_full[st], (it >> 1) & 1);   // implies both Y stages are resident (their S' MMAs ran before the dS warps did)
        tc_fence_after();
        const uint32_t tA = tmem_base + COL_DS + st * 64;
        const uint32_t acc = it > 0;
        if (elect_one()) {
          if (G2) {
            const uint64_t b = dm2 + uint64_t((s2 * Y2_STAGE) >> 4);
#pragma unroll
            for (int k = 0; k < 4; ++k) umma_bf16_ts(tmem_base + COL_DX2, tA + 32 + k * 8, b + uint64_t((k * 2048) >> 4), idesc_g2, acc | (k != 0));
            umma_commit(&y2_empty[s2]);
          }
          if (G1) {
            const uint64_t b = dm1 + uint64_t((s1 * Y1_STAGE) >> 4);
#pragma unroll
            for (int k = 0; k < 4; ++k) umma_bf16_ts(tmem_base + COL_DX1, tA + k * 8, b + uint64_t((k * 2048) >> 4), idesc_g1, acc | (k != 0));
            umma_commit(&y1_empty[s1]);
          }
          umma_commit(&ds_empty[st]);
          if (it + 1 == nsteps) umma_commit(dx_full);
        }
        __syncwarp();
        if (++s1 == NS1) s1 = 0;
        if (++s2 == NS2) s2 = 0;
      }
    }
  } else {
    // ===================== dS warps =====================
    reg_alloc<112>();
    const int sw = warp - 4;
    const int quarter = warp & 3;
    const int grp = sw >> 2;
    const int par = grp & 1;
    const int half = grp >> 1;
    const int rloc = quarter * 32 + lane;
    const int xrow = x0 + rloc;
    const float L2E = 1.4426950408889634f, LN2 = 0.6931471805599453f;
    const float sc1 = p.c1 * L2E, sc2 = p.c2 * L2E;
    float nL1 = -1e30f, nL2 = -1e30f, klog = 0.f, my_g = 0.f;
    if (!OWNER_K && xrow < p.NQ) {
      const float* sp = reinterpret_cast<const float*>(p.stats + (size_t(unit) * NQP + size_t(xrow & ~1)));
      const int u = xrow & 1;
      nL1 = sp[u]; nL2 = sp[2 + u]; my_g = sp[4 + u]; klog = sp[6 + u];
    }
    const uint32_t lane_addr = tmem_base + (uint32_t(quarter * 32) << 16);
    const uint32_t stat_base = smem_u32(sStat) + half * 32 * 16;
    const uint32_t ds_addr = lane_addr + COL_DS + par * 64 + half * 16;
    const bool f16 = p.fmt16 == 0, relu2 = p.act2 == 1;
    for (int it = par; it < nsteps; it += 2) {
      const int j = step_j(it);
      const int ss = it % NSS;
      mbar_wait(&s_full[par], (it >> 1) & 1);
      tc_fence_after();
      const uint32_t taddr = lane_addr + ss * 128 + half * 32;
      uint32_t r1[32], r2[32], o1[16], o2[16];
      tmem_ld32(taddr, r1);
      tmem_ld32(taddr + 64, r2);
      tmem_wait_ld();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&s_empty[par]);
      const int y0 = j * C::BY + half * 32;
      const bool masked = OWNER_K ? (CAUSAL && (y0 + off < x0 + C::BX - 1))
                                  : ((CAUSAL && (y0 + 31 > x0 + off)) || (y0 + 32 > p.NK));
      const uint32_t stat = stat_base + (it % NST) * C::STAT_STAGE;
      dispatch3(masked, f16, relu2, [&](auto m, auto h, auto r) {
        ds_row<32, G1, OWNER_K, CAUSAL, decltype(m)::value, G2, decltype(h)::value, decltype(r)::value>(
            r1, r2, o1, o2, sc1, sc2, nL1, nL2, klog, stat, xrow, y0, off, p.NK);
      });
      mbar_wait(&ds_empty[par], ((it >> 1) & 1) ^ 1);
      tc_fence_after();
      if (G2) tmem_st16(ds_addr + 32, o2);
      if (G1) tmem_st16(ds_addr, o1);
      tmem_wait_st();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&ds_full[par]);
    }
    // ---- epilogue: each warp group takes a quarter of the (padded) columns, 16 at a time
    const bool valid = xrow < NX;
    const long long xr = valid ? xrow : 0;
    const float g_row = OWNER_K ? 1.f : my_g;
    auto store_all = [&](uint16_t* base, const OutGeom& g, int D, uint32_t col_dx, float scale) {
      const int c0 = grp * (D / 4);
      uint16_t* o = base + (bx * g.sb + hx * g.sh + xr * g.sn) + c0;
      if (nsteps > 0) {
        for (int c = 0; c < D / 4; c += 16) store_dx_cols<16>(lane_addr + col_dx + c0 + c, scale, o + c, valid, f16, c0 + c, g.d);
      } else if (valid) {
        const uint4 z = make_uint4(0, 0, 0, 0);
        for (int c = 0; c < D / 4 && c0 + c < g.d; c += 8) *reinterpret_cast<uint4*>(o + c) = z;
      }
    };
    if (nsteps > 0) {
      mbar_wait(dx_full, 0);
      tc_fence_after();
    }
    if (G2) store_all(p.dX2, p.g2, D2, COL_DX2, p.c2 * g_row);
    if (G1) store_all(p.dX1, p.g1, D1, COL_DX1, p.c1 * LN2 * g_row);
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 2) {
    tc_fence_after();
    tmem_dealloc<C::TMEM_COLS>(tmem_base);
  }
}

}  // namespace skl
