// streamkl_bwd_fused_sm100.cuh -- one-visit ("fused") StreamKL backward: the CTA owns a 128-row K tile,
// visits every (query tile, key tile) pair ONCE, accumulates dK in place and adds its dQ contribution with fp32 atomics.
// One pass per differentiated distribution: the student pass (TPASS = false: dS2 -> dK2, dQ2; all of Setting 1) and the
// teacher pass (TPASS = true: dS1 -> dK1, dQ1; Setting 2 runs both).  Against the separate kernels (streamkl_bwd_sm100.cuh)
// the student pass alone halves the logit recomputation and the exps of Setting 1; for Setting 2 the two passes execute the
// same work as the two owner kernels, but both grids are K-owner grids (bsz x T_K CTAs), which is what fills the machine
// when N_Q is small.  The price is an fp32 dQ workspace, a convert pass, and a dQ that is reproducible only up to fp32
// summation order (the separate kernels remain the deterministic mode).  Below, "2" stands for the pass's distribution.
//
// Per 64-query step, with K = the owned key tile (X) and Q = the streamed query tile (Y):
//   S1' = K1 Q1^T, S2' = K2 Q2^T          tcgen05.mma (SS) -> TMEM, lane = key                                   (B2)
//   dS2 = g (P2 - P1)                      dS warps, as in the K-owner kernel (B3, B4), written twice:
//                                            packed bf16 into TMEM  (A operand of the dK2 product) and
//                                            into swizzled shared memory [key][query] (B operand of the dQ2 product;
//                                            B cannot come from TMEM)
//   dK2  += dS2 Q2                          tcgen05.mma, A from TMEM, B = Q2 tile read MN-major
//   dQ2^T = K2^T dS2                        tcgen05.mma, A = K2 tile read MN-major, B = dS2 tile read MN-major,
//                                            M = d2 (padded to 128), N = 64 queries, K = 128 keys -> a TMEM stage of
//                                            [d][query] fp32, drained by the dS warps with red.global.add.f32 into the
//                                            fp32 workspace (a warp's 32 lanes = 32 consecutive d: one 128-byte line)
// TMEM (512 columns): NSS x {S1' 64, S2' 64} | 2 x dS2 32 | dK2 D2 | 2 x dQ2^T 64.
#pragma once
#include "streamkl_bwd_sm100.cuh"

namespace skl {

template <int D1, int D2, bool TPASS = false>
struct BwdFusedCfg {
  static_assert(D1 % 64 == 0 && D2 % 64 == 0 && D1 <= 128 && D2 <= 128, "tcgen05 path: d in {64,128}");
  static constexpr int BX = 128, BY = 64;
  static constexpr int KB1 = D1 / 64, KB2 = D2 / 64;
  static constexpr int XBLK = BX * 128, YBLK = BY * 128;
  static constexpr int X_BYTES = (KB1 + KB2) * XBLK;
  static constexpr int DS_TILE = BX * BY * 2;                 // [128 keys x 64 queries] bf16, 128-byte rows, SW128
  static constexpr int DS_BYTES = 2 * DS_TILE;
  static constexpr int Y_STAGE = (KB1 + KB2) * YBLK;
  static constexpr int STAT_STAGE = BY * 16;
  static constexpr int AUX_BYTES = 512;
  static constexpr int NSTAGE_RAW = (227 * 1024 - 1024 - AUX_BYTES - X_BYTES - DS_BYTES) / (Y_STAGE + STAT_STAGE);
  static constexpr int NSTAGE = NSTAGE_RAW > 6 ? 6 : NSTAGE_RAW;
  static_assert(NSTAGE >= 2, "need at least a double-buffered Y ring");
  static constexpr int SMEM_BYTES = 1024 + X_BYTES + DS_BYTES + NSTAGE * (Y_STAGE + STAT_STAGE) + AUX_BYTES;
  static constexpr int THREADS = 128 + 512;
  static constexpr uint32_t TMEM_COLS = 512;
  static constexpr int DG = TPASS ? D1 : D2;                  // head dim of the distribution this pass differentiates
  static constexpr int NSS = (512 - 64 - DG - 128) / 128 >= 2 ? 2 : 1;
  static constexpr uint32_t COL_DS = NSS * 128;               // 2 stages x 32 packed columns
  static constexpr uint32_t COL_DK = COL_DS + 64;
  static constexpr uint32_t COL_DQ = COL_DK + DG;             // 2 stages x 64 columns (queries), lane = d
  static_assert(COL_DQ + 128 <= 512, "TMEM budget");
};

struct BwdFusedParams {
  int NQ, NK, TX, BH;    // BH = B * H query heads
  int H, HK, G;          // query heads, K heads, query heads per K head (GQA)
  uint32_t fmt16;        // 1 bf16, 0 fp16
  int act2;              // student activation: 0 none, 1 relu (R23)
  float c1, c2;
  const float4* stats;   // as BwdParams::stats
  float* dq_acc;         // [BH][NQ][DG] fp32, zeroed by the caller of the kernel
  uint16_t* dK;          // dK2 (student pass) or dK1 (teacher pass), 16-bit elements
  OutGeom gk;            // its strides and true head dim
};

// dQ = 16-bit(scale * dq_acc): the one rounding of the atomically accumulated gradient (scale = c2, or c1 ln2 for the teacher).
// dq_acc is dense [B*H][NQ][DG] (DG = padded head dim); dQ has the caller's strides and true head dim.  One thread per 4 columns.
__global__ void streamkl_bwd_dq_convert_kernel(const float4* __restrict__ acc, uint16_t* __restrict__ out, float scale, long long n4,
                                               int NQ, int H, int DG, OutGeom g, int f16) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n4) return;
  const int c4 = DG / 4;
  const int col = int(i % c4) * 4;
  if (col >= g.d) return;
  const long long r = i / c4;
  const int row = int(r % NQ);
  const long long bh = r / NQ;
  const float4 v = acc[i];
  uint16_t* o = out + (bh / H) * g.sb + (bh % H) * g.sh + (long long)row * g.sn + col;
  *reinterpret_cast<uint2*>(o) = f16 ? make_uint2(pack_f16x2(v.x * scale, v.y * scale), pack_f16x2(v.z * scale, v.w * scale))
                                     : make_uint2(pack_bf16x2(v.x * scale, v.y * scale), pack_bf16x2(v.z * scale, v.w * scale));
}

template <int D1, int D2, bool CAUSAL, bool TPASS = false>
__global__ void __launch_bounds__(BwdFusedCfg<D1, D2, TPASS>::THREADS, 1)
streamkl_bwd_fused_sm100_kernel(const __grid_constant__ CUtensorMap tmQ1, const __grid_constant__ CUtensorMap tmK1,
                                const __grid_constant__ CUtensorMap tmQ2, const __grid_constant__ CUtensorMap tmK2,
                                const BwdFusedParams p) {
  using C = BwdFusedCfg<D1, D2, TPASS>;
  constexpr int DG = C::DG;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t* sX1 = smem;                                    // K1 tile (owner)
  uint8_t* sX2 = sX1 + C::KB1 * C::XBLK;                  // K2 tile
  uint8_t* sDS = smem + C::X_BYTES;                       // 2 x dS2 tile [key][query]
  uint8_t* sY = sDS + C::DS_BYTES;                        // NSTAGE x {Q1 blocks, Q2 blocks}
  float4* sStat = reinterpret_cast<float4*>(sY + C::NSTAGE * C::Y_STAGE);
  uint64_t* bars = reinterpret_cast<uint64_t*>(reinterpret_cast<uint8_t*>(sStat) + C::NSTAGE * C::STAT_STAGE);
  uint64_t* x_full = bars;                       // 1
  uint64_t* y_full = bars + 1;                   // NSTAGE
  uint64_t* y_empty = y_full + C::NSTAGE;        // NSTAGE (count 2: S' MMAs and dK2 MMAs)
  uint64_t* s_full = y_empty + C::NSTAGE;        // 2 per parity group
  uint64_t* s_empty = s_full + 2;                // 2 (8 warps)
  uint64_t* ds_full = s_empty + 2;               // 2 (8 warps): dS2 of the group's step is in TMEM and in shared memory
  uint64_t* ds_empty = ds_full + 2;              // 2 (1): the dK2 and dQ2 MMAs that read it have retired
  uint64_t* dq_full = ds_empty + 2;              // 2 (1): dQ2^T stage written by the tensor pipe
  uint64_t* dq_empty = dq_full + 2;              // 2 (8 warps): drained to registers
  uint64_t* dk_full = dq_empty + 2;              // 1
  uint32_t* tmem_ptr = reinterpret_cast<uint32_t*>(dk_full + 1);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int unit = blockIdx.x / p.TX;            // (batch, K head); the query tiles of its G query heads are streamed in turn
  const int bx = unit / p.HK, hx = unit % p.HK;
  const int xt = blockIdx.x % p.TX;              // early K tiles are seen by more queries: heavy first
  const int x0 = xt * C::BX;
  const int off = p.NK - p.NQ;
  const long long NQP = bwd_stats_padded_rows(p.NQ);
  int j_begin = 0;
  const int j_end = (p.NQ + C::BY - 1) / C::BY;
  if (CAUSAL) j_begin = max(0, x0 - off) / C::BY;    // first query that sees key x0
  const int nsteps1 = max(0, j_end - j_begin);   // steps per streamed query head
  const int nsteps = nsteps1 * p.G;
  auto step_g = [&](int it) { return it / max(nsteps1, 1); };
  auto step_j = [&](int it) { return j_begin + it % max(nsteps1, 1); };

  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tmQ1); tma_prefetch_desc(&tmK1); tma_prefetch_desc(&tmQ2); tma_prefetch_desc(&tmK2);
  }
  if (warp == 1 && lane == 0) {
    mbar_init(x_full, 1);
    for (int s = 0; s < C::NSTAGE; ++s) { mbar_init(&y_full[s], 1); mbar_init(&y_empty[s], 2); }
    for (int w = 0; w < 2; ++w) {
      mbar_init(&s_full[w], 1); mbar_init(&s_empty[w], 8);
      mbar_init(&ds_full[w], 8); mbar_init(&ds_empty[w], 1);
      mbar_init(&dq_full[w], 1); mbar_init(&dq_empty[w], 8);
    }
    mbar_init(dk_full, 1);
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
        mbar_arrive_expect_tx(x_full, C::X_BYTES);
#pragma unroll
        for (int kb = 0; kb < C::KB1; ++kb) tma_load_4d_hint(sX1 + kb * C::XBLK, &tmK1, x_full, kb * 64, x0, hx, bx, pol_x);
#pragma unroll
        for (int kb = 0; kb < C::KB2; ++kb) tma_load_4d_hint(sX2 + kb * C::XBLK, &tmK2, x_full, kb * 64, x0, hx, bx, pol_x);
        for (int it = 0; it < nsteps; ++it) {
          const int j = step_j(it);
          const int hy = hx * p.G + step_g(it);        // streamed query head
          const int s = it % C::NSTAGE;
          mbar_wait(&y_empty[s], ((it / C::NSTAGE) & 1) ^ 1);
          mbar_arrive_expect_tx(&y_full[s], C::Y_STAGE + C::STAT_STAGE);
          uint8_t* st = sY + s * C::Y_STAGE;
#pragma unroll
          for (int kb = 0; kb < C::KB1; ++kb) tma_load_4d_hint(st + kb * C::YBLK, &tmQ1, &y_full[s], kb * 64, j * C::BY, hy, bx, pol_y);
#pragma unroll
          for (int kb = 0; kb < C::KB2; ++kb)
            tma_load_4d_hint(st + (C::KB1 + kb) * C::YBLK, &tmQ2, &y_full[s], kb * 64, j * C::BY, hy, bx, pol_y);
          bulk_load_1d(sStat + s * C::BY, p.stats + (size_t(bx * p.H + hy) * NQP + size_t(j) * C::BY), C::STAT_STAGE, &y_full[s]);
        }
      }
    } else if (warp == 1) {
      // ===================== S' MMA issuer =====================
      const uint32_t idesc_s = umma_idesc_16(C::BX, C::BY, 0, 0, p.fmt16);
      const uint64_t dx1 = umma_smem_desc_sw128(smem_u32(sX1), 16, 1024);
      const uint64_t dx2 = umma_smem_desc_sw128(smem_u32(sX2), 16, 1024);
      const uint64_t dyk = umma_smem_desc_sw128(smem_u32(sY), 16, 1024);
      if (nsteps > 0) {
        mbar_wait(x_full, 0);
        tc_fence_after();
      }
      for (int it = 0; it < nsteps; ++it) {
        const int s = it % C::NSTAGE;
        const int ss = it % C::NSS;
        const int prev = it - C::NSS;
        mbar_wait(&y_full[s], (it / C::NSTAGE) & 1);
        if (prev >= 0) mbar_wait(&s_empty[prev & 1], (prev >> 1) & 1);
        tc_fence_after();
        uint64_t dys = dyk + uint64_t((s * C::Y_STAGE) >> 4), a1 = dx1, a2 = dx2;
        asm volatile("" : "+l"(a1), "+l"(a2), "+l"(dys));   // descriptors = base + immediate (see streamkl_bwd_sm100.cuh)
        const uint32_t tS1 = tmem_base + ss * 128, tS2 = tS1 + 64;
        if (elect_one()) {
#pragma unroll
          for (int kb = 0; kb < C::KB1; ++kb)
#pragma unroll
            for (int k = 0; k < 4; ++k)
              umma_bf16_ss(tS1, a1 + uint64_t((kb * C::XBLK + k * 32) >> 4), dys + uint64_t((kb * C::YBLK + k * 32) >> 4), idesc_s,
                           (kb | k) != 0);
#pragma unroll
          for (int kb = 0; kb < C::KB2; ++kb)
#pragma unroll
            for (int k = 0; k < 4; ++k)
              umma_bf16_ss(tS2, a2 + uint64_t((kb * C::XBLK + k * 32) >> 4),
                           dys + uint64_t(((C::KB1 + kb) * C::YBLK + k * 32) >> 4), idesc_s, (kb | k) != 0);
          umma_commit(&s_full[it & 1]);
          umma_commit(&y_empty[s]);
        }
        __syncwarp();
      }
    } else if (warp == 3) {
      // ===================== gradient MMA issuer =====================
      const uint32_t idesc_k = umma_idesc_16(C::BX, DG, 0, 1, p.fmt16);    // dK2 += dS2 Q2   : A from TMEM, B = Q2 MN-major
      const uint32_t idesc_q = umma_idesc_16(128, C::BY, 1, 1, p.fmt16);   // dQ2^T = K2^T dS2: A = K2 MN-major, B = dS2 MN-major
      // MN-major operands: rows = the contraction index (128 B each, 8-row groups 1024 B apart = SBO), 64-element chunks
      // of the M/N index LBO bytes apart; a K=16 slice = 16 rows = 2048 B.  For d2 = 64 the padded half of M reads the
      // shared memory behind the K2 tile: those accumulator lanes (d >= 64) are never drained.
      const uint64_t dym = umma_smem_desc_sw128(smem_u32(sY), C::YBLK, 1024);
      const uint64_t dka = umma_smem_desc_sw128(smem_u32(TPASS ? sX1 : sX2), C::XBLK, 1024);
      const uint64_t dsb = umma_smem_desc_sw128(smem_u32(sDS), C::DS_TILE, 1024);
      for (int it = 0; it < nsteps; ++it) {
        const int s = it % C::NSTAGE;
        const int par = it & 1;
        const uint32_t u = uint32_t(it >> 1);
        mbar_wait(&ds_full[par], u & 1);
        mbar_wait(&dq_empty[par], (u & 1) ^ 1);     // the dQ2^T stage of step it-2 has been copied to registers
        tc_fence_after();
        uint64_t dys = dym + uint64_t((s * C::Y_STAGE + (TPASS ? 0 : C::KB1 * C::YBLK)) >> 4), ka = dka, db = dsb + uint64_t((par * C::DS_TILE) >> 4);
        asm volatile("" : "+l"(dys), "+l"(ka), "+l"(db));
        const uint32_t tA = tmem_base + C::COL_DS + par * 32;
        const uint32_t acc = it > 0;
        if (elect_one()) {
#pragma unroll
          for (int k = 0; k < 4; ++k)      // K = 64 queries
            umma_bf16_ts(tmem_base + C::COL_DK, tA + k * 8, dys + uint64_t((k * 2048) >> 4), idesc_k, acc | (k != 0));
#pragma unroll
          for (int k = 0; k < 8; ++k)      // K = 128 keys
            umma_bf16_ss(tmem_base + C::COL_DQ + par * 64, ka + uint64_t((k * 2048) >> 4), db + uint64_t((k * 2048) >> 4), idesc_q,
                         k != 0);
          umma_commit(&ds_empty[par]);
          umma_commit(&y_empty[s]);
          umma_commit(&dq_full[par]);
          if (it + 1 == nsteps) umma_commit(dk_full);
        }
        __syncwarp();
      }
    }
  } else {
    // ===================== dS warps =====================
    reg_alloc<112>();
    const int sw = warp - 4;
    const int quarter = warp & 3;
    const int grp = sw >> 2;
    const int par = grp & 1;                  // step parity this group serves (= its dS2 and dQ2^T stage)
    const int half = grp >> 1;                // 32-query half of every streamed tile
    const int rloc = quarter * 32 + lane;     // key row within the tile = TMEM lane (= d index when draining dQ2^T)
    const int xrow = x0 + rloc;
    const float L2E = 1.4426950408889634f;
    const float sc1 = p.c1 * L2E, sc2 = p.c2 * L2E;
    const uint32_t lane_addr = tmem_base + (uint32_t(quarter * 32) << 16);
    const uint32_t stat_base = smem_u32(sStat) + half * 32 * 16;
    const uint32_t ds_taddr = lane_addr + C::COL_DS + par * 32 + half * 16;
    uint8_t* ds_srow = sDS + par * C::DS_TILE + rloc * 128;
    const int swz = rloc & 7;
    const uint32_t dq_taddr = lane_addr + C::COL_DQ + par * 64 + half * 32;
    const bool d_valid = rloc < DG;           // this lane's d index exists (d = 64: lanes 64..127 are padding)

    // copy the dQ2^T stage of step `itd` (one of this group's steps) to registers, free the stage, add it to the fp32 workspace
    auto drain = [&](int itd) {
      mbar_wait(&dq_full[par], (itd >> 1) & 1);
      tc_fence_after();
      uint32_t q[32];
      tmem_ld32(dq_taddr, q);
      tmem_wait_ld();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&dq_empty[par]);
      if (d_valid) {
        const int q0 = step_j(itd) * C::BY + half * 32;
        float* dst = p.dq_acc + (size_t(bx * p.H + hx * p.G + step_g(itd)) * p.NQ + q0) * DG + rloc;
#pragma unroll
        for (int c = 0; c < 32; ++c)
          if (q0 + c < p.NQ) atomicAdd(dst + size_t(c) * DG, __uint_as_float(q[c]));   // result unused: red.global.add.f32
      }
    };

    int last = -1;
    const bool f16 = p.fmt16 == 0, relu2 = p.act2 == 1;
    for (int it = par; it < nsteps; it += 2) {
      const int j = step_j(it);
      const int s = it % C::NSTAGE;
      const int ss = it % C::NSS;
      const uint32_t u = uint32_t(it >> 1);
      mbar_wait(&s_full[par], u & 1);
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
      // warp-uniform: causal diagonal blocks, and the owner tile's KEY tail (TMA zero-fills those rows, P = exp2(0 - lse) may
      // be inf there, and unlike the separate K-owner kernel this kernel CONTRACTS over the owned keys: dQ2^T = K2^T dS2)
      const bool masked = (CAUSAL && (y0 + off < x0 + C::BX - 1)) || (x0 + C::BX > p.NK);
      const uint32_t stat = stat_base + s * C::STAT_STAGE;
      // (o2 = the pass's dS: the teacher pass takes ds_row's dS1 output)
      uint32_t (&f1)[16] = *(TPASS ? &o2 : &o1), (&f2)[16] = *(TPASS ? &o1 : &o2);
      dispatch3(masked, f16, relu2, [&](auto m, auto h, auto r) {
        ds_row<32, TPASS, true, CAUSAL, decltype(m)::value, !TPASS, decltype(h)::value, decltype(r)::value>(
            r1, r2, f1, f2, sc1, sc2, 0.f, 0.f, 0.f, stat, xrow, y0, off, p.NK);
      });
      // the previous step of this group: its dQ2^T MMAs were issued when the group signalled ds_full and have had this step's
      // whole dS computation to finish (draining right after the logit load stalled ~600 cycles per step on dq_full: ncu)
      if (last >= 0) drain(last);
      mbar_wait(&ds_empty[par], (u & 1) ^ 1);   // the MMAs of step it-2 have consumed both copies of this dS2 stage
      tc_fence_after();
      tmem_st16(ds_taddr, o2);
#pragma unroll
      for (int c = 0; c < 4; ++c)               // [key][query] tile, 128-byte rows, 16-byte chunk index XOR (row mod 8)
        *reinterpret_cast<uint4*>(ds_srow + (((half * 4 + c) ^ swz) << 4)) = make_uint4(o2[4 * c], o2[4 * c + 1], o2[4 * c + 2], o2[4 * c + 3]);
      fence_proxy_async_smem();
      tmem_wait_st();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&ds_full[par]);
      last = it;
    }
    if (last >= 0) drain(last);
    // ---- epilogue: dK (TMEM fp32) * scale -> 16-bit -> HBM; each warp group takes a quarter of the (padded) columns
    const bool valid = xrow < p.NK;
    uint16_t* ok = p.dK + (bx * p.gk.sb + hx * p.gk.sh + (long long)(valid ? xrow : 0) * p.gk.sn) + grp * (DG / 4);
    if (nsteps > 0) {
      mbar_wait(dk_full, 0);
      tc_fence_after();
      // (the teacher's dS1 is kept in log2 units, Eq.12: its ln2 joins the scale here, as in the separate kernels)
      store_dx_cols<DG / 4>(lane_addr + C::COL_DK + grp * (DG / 4), TPASS ? p.c1 * 0.6931471805599453f : p.c2, ok, valid, f16,
                            grp * (DG / 4), p.gk.d);
    } else if (valid) {
      const uint4 z = make_uint4(0, 0, 0, 0);
      for (int c = 0; c < DG / 4 && grp * (DG / 4) + c < p.gk.d; c += 8) *reinterpret_cast<uint4*>(ok + c) = z;
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
