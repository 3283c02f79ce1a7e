// streamkl_fwd_sm100.cuh -- StreamKL forward (Algorithm 1) for sm_100a.
//
// One CTA owns NMT 128-row M-tiles of one (b,h) and streams BK-key tiles, NMT * BK = 128 (STREAMKL_FWD_BK = 128: one
// M-tile, 128-key steps, N=128 logit MMAs -- the default; 64: two M-tiles sharing 64-key tiles):
//   warp 0      TMA producer : Q1,Q2 once; K1_j,K2_j through an NSTAGE ring          (F1, F2 of DESIGN.md)
//   warp 1      MMA issuer   : S1 = Q1 K1_j^T, S2 = Q2 K2_j^T, tcgen05.mma -> TMEM    (F3)
//   warp 2      TMEM allocator
//   warps 4-19  sixteen softmax warps = NMT M-tiles x BK/32 column groups x 4 TMEM lane quarters    (F4, F5, F6)
// TMEM (512 columns): per M-tile two stages of {S1 (BK cols), S2 (BK cols)}.  A softmax thread owns ONE query row and
// ONE 32-column group of every key tile: it pulls its 32+32 logits into registers, releases the TMEM stage at once (so
// the next tile's MMA overlaps the exp work) and performs the online update of its own partial (m1,l1,m2,l2,acc) --
// Eq.9-10 -- entirely thread-locally in the log2 domain (exp2 instead of exp; R6).  The
// column groups of a row are independent partial statistics over disjoint key sets; they are merged once, after the
// last tile, with the associative merge of Eq.11 (carrying (m2,l2) too: R11).  Four softmax warps per
// SM sub-partition keep the MUFU pipe fed while other warps sit in their no-exp phases (TMEM load, barrier waits).
#pragma once
#include <cuda_bf16.h>
#include <math_constants.h>

#include "sm100_ptx.cuh"

// Share of the forward's exps evaluated by the FMA-pipe polynomial (ex2_poly2): one column pair in every
// STREAMKL_FWD_POLY_EVERY (0 = none).  The forward is MUFU-bound 2:1 against the tensor pipe.
#ifndef STREAMKL_FWD_POLY_EVERY
#define STREAMKL_FWD_POLY_EVERY 4
#endif

// 1: unmasked tiles are evaluated against the row's current reference and the row maximum is only recomputed when a
// tile sum shows the reference is stale (online_update_lazy); 0: Alg.1 literally (row maximum every tile).
// Keys per step = N of the logit MMAs.  64: two 128-row M-tiles per CTA share every K tile (half the L2->SM traffic), but
// an N=64 SS MMA is shared-memory-bound at 48 cycles instead of 32.  128: one M-tile per CTA, N=128 MMAs at
// the full tensor rate.
#ifndef STREAMKL_FWD_BK
#define STREAMKL_FWD_BK 128
#endif

#ifndef STREAMKL_FWD_LAZY_MAX
#define STREAMKL_FWD_LAZY_MAX 1
#endif

namespace skl {

template <int D1, int D2>
struct FwdCfg {
  static_assert(D1 % 64 == 0 && D2 % 64 == 0 && D1 <= 128 && D2 <= 128, "tcgen05 path: d in {64,128}");
  static constexpr int BM = 128;             // rows per M-tile (TMEM lanes)
  static constexpr int BK = STREAMKL_FWD_BK; // keys per step = N of the logit MMAs
  static_assert(BK == 64 || BK == 128, "TMEM holds 2 stages x {S1,S2} x BK columns for NMT M-tiles: NMT * BK = 128");
  static constexpr int NMT = 128 / BK;       // M-tiles per CTA
  static constexpr int BQ = BM * NMT;        // query rows per CTA
  static constexpr int KB1 = D1 / 64, KB2 = D2 / 64;  // 128-byte K-blocks per row
  static constexpr int QBLK = BM * 128;      // bytes of one [128 rows x 64 bf16] swizzled block
  static constexpr int KBLK = BK * 128;      // bytes of one [64 rows x 64 bf16] swizzled block
  static constexpr int Q_BYTES = NMT * (KB1 + KB2) * QBLK;
  static constexpr int STAGE_BYTES = (KB1 + KB2) * KBLK;
  static constexpr int SMEM_LIMIT = 227 * 1024;
  static constexpr int AUX_BYTES = 256;      // barriers + tmem pointer
  static constexpr int NSTAGE_RAW = (SMEM_LIMIT - 1024 - AUX_BYTES - Q_BYTES) / STAGE_BYTES;
  static constexpr int NSTAGE = NSTAGE_RAW > 6 ? 6 : NSTAGE_RAW;
  static_assert(NSTAGE >= 2, "need at least a double-buffered K ring");
  static constexpr int SMEM_BYTES = 1024 + Q_BYTES + NSTAGE * STAGE_BYTES + AUX_BYTES;
  static constexpr int NHALF = BK / 32;      // column groups of a key tile (one softmax thread per row and group)
  static constexpr int BC = BK / NHALF;      // columns per softmax thread and step (32)
  static constexpr int THREADS = 128 + NMT * NHALF * 128;
  static_assert(THREADS == 640, "sixteen softmax warps");
  static constexpr uint32_t TMEM_COLS = 512;
};

struct FwdParams {
  int NQ, NK, TQ;       // TQ = number of BQ-row CTA tiles per head
  int BH;
  float sc1, sc2;       // c_t * log2(e)
  float* kl;
  float* lse1;
  float* lse2;
  // split-K: W contiguous key chunks of `chunk_steps` 64-key steps each; partial statistics
  // (m1,l1,m2,l2,acc in the log2 domain) go to part[bh][w][5][NQ] and streamkl_fwd_splitk_reduce_kernel merges them
  int W, chunk_steps;
  float* part;
};

// Online update for NC keys of one query row (thread-local).  Implements Alg.1 lines 8-12 with
//   x_t = s_t*sc_t - m_t (log2 domain, shifted),  acc += sum p1*(x1-x2) + (m1-m2)*sum p1   [= sum p1 (s1'-s2')].
struct RowState {
  float m1, m2, l1, l2, acc;
};

template <bool MASKED, int NC>
__device__ __forceinline__ void online_update(RowState& st, const uint32_t (&r1)[NC], const uint32_t (&r2)[NC], float sc1,
                                              float sc2, int kbase, int limit) {
  float mx1a = -CUDART_INF_F, mx1b = -CUDART_INF_F, mx2a = -CUDART_INF_F, mx2b = -CUDART_INF_F;
  if constexpr (!MASKED) {
#pragma unroll
    for (int e = 0; e < NC; e += 4) {
      mx1a = max3(mx1a, __uint_as_float(r1[e]), __uint_as_float(r1[e + 1]));
      mx1b = max3(mx1b, __uint_as_float(r1[e + 2]), __uint_as_float(r1[e + 3]));
      mx2a = max3(mx2a, __uint_as_float(r2[e]), __uint_as_float(r2[e + 1]));
      mx2b = max3(mx2b, __uint_as_float(r2[e + 2]), __uint_as_float(r2[e + 3]));
    }
  } else {
#pragma unroll
    for (int e = 0; e < NC; ++e) {
      const bool ok = (kbase + e) <= limit;
      mx1a = fmaxf(mx1a, ok ? __uint_as_float(r1[e]) : -CUDART_INF_F);
      mx2a = fmaxf(mx2a, ok ? __uint_as_float(r2[e]) : -CUDART_INF_F);
    }
  }
  const float m1n = fmaxf(st.m1, fmaxf(mx1a, mx1b) * sc1);  // sc > 0: max commutes with the scale
  const float m2n = fmaxf(st.m2, fmaxf(mx2a, mx2b) * sc2);
  // R7: a row whose every key so far is masked keeps m = -inf; use reference 0 so (-inf)-(-inf) never forms
  const float ref1 = MASKED ? (m1n == -CUDART_INF_F ? 0.f : m1n) : m1n;
  const float ref2 = MASKED ? (m2n == -CUDART_INF_F ? 0.f : m2n) : m2n;
  const float a1 = ex2_approx(st.m1 - ref1);  // alpha_1 (Alg.1 line 9); m = -inf gives 0
  const float a2 = ex2_approx(st.m2 - ref2);
  float sum1, sum2, dsum;
  if constexpr (!MASKED) {
    // packed fp32x2 lanes over column pairs (e, e+1): half the issue slots of the scalar form (the loop is
    // issue/MUFU bound); two independent accumulator pairs per quantity
    const float2 vsc1 = make_float2(sc1, sc1), vsc2 = make_float2(sc2, sc2);
    const float2 vr1 = make_float2(-ref1, -ref1), vr2 = make_float2(-ref2, -ref2);
    float2 s1v[2] = {make_float2(0.f, 0.f), make_float2(0.f, 0.f)}, s2v[2] = {s1v[0], s1v[0]}, ddv[2] = {s1v[0], s1v[0]};
#pragma unroll
    for (int e = 0; e < NC; e += 2) {
      const float2 x1 = fma2(make_float2(__uint_as_float(r1[e]), __uint_as_float(r1[e + 1])), vsc1, vr1);
      const float2 x2 = fma2(make_float2(__uint_as_float(r2[e]), __uint_as_float(r2[e + 1])), vsc2, vr2);
      // every STREAMKL_FWD_POLY_EVERY-th column pair takes its two exps on the FMA/ALU pipes instead of MUFU
      const bool poly = STREAMKL_FWD_POLY_EVERY > 0 && ((e >> 1) % (STREAMKL_FWD_POLY_EVERY > 0 ? STREAMKL_FWD_POLY_EVERY : 1)) == 0;
      const float2 p1 = poly ? ex2_poly2(x1) : make_float2(ex2_approx(x1.x), ex2_approx(x1.y));
      const float2 p2 = poly ? ex2_poly2(x2) : make_float2(ex2_approx(x2.x), ex2_approx(x2.y));
      const int a = (e >> 1) & 1;
      s1v[a] = add2(s1v[a], p1);
      s2v[a] = add2(s2v[a], p2);
      ddv[a] = fma2(p1, sub2(x1, x2), ddv[a]);
    }
    sum1 = (s1v[0].x + s1v[0].y) + (s1v[1].x + s1v[1].y);
    sum2 = (s2v[0].x + s2v[0].y) + (s2v[1].x + s2v[1].y);
    dsum = (ddv[0].x + ddv[0].y) + (ddv[1].x + ddv[1].y);
  } else {
    float s1[4] = {0.f, 0.f, 0.f, 0.f}, s2[4] = {0.f, 0.f, 0.f, 0.f}, dd[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
    for (int e = 0; e < NC; ++e) {
      const float x1 = fmaf(__uint_as_float(r1[e]), sc1, -ref1);
      const float x2 = fmaf(__uint_as_float(r2[e]), sc2, -ref2);
      // R8: zero P~ at masked entries, take the difference from the raw (finite) logits
      const bool ok = (kbase + e) <= limit;
      const float p1 = ok ? ex2_approx(x1) : 0.f;
      const float p2 = ok ? ex2_approx(x2) : 0.f;
      s1[e & 3] += p1;
      s2[e & 3] += p2;
      dd[e & 3] = fmaf(p1, x1 - x2, dd[e & 3]);
    }
    sum1 = (s1[0] + s1[1]) + (s1[2] + s1[3]);
    sum2 = (s2[0] + s2[1]) + (s2[2] + s2[3]);
    dsum = (dd[0] + dd[1]) + (dd[2] + dd[3]);
  }
  st.l1 = fmaf(st.l1, a1, sum1);                               // line 11 (R9: alpha1 on l1, acc; alpha2 on l2)
  st.l2 = fmaf(st.l2, a2, sum2);
  st.acc = fmaf(st.acc, a1, fmaf(ref1 - ref2, sum1, dsum));    // line 12
  st.m1 = m1n;
  st.m2 = m2n;
}

// Unmasked tiles, lazy reference.  Alg.1 keeps m_t = the running MAXIMUM, but Eq.8-10 hold for ANY per-row reference
// m_t as long as (l_t, acc) are expressed relative to it: the maximum is only there to keep exp() in range.  So the tile
// is first evaluated against the reference the row already has -- no row-max reduction, no alpha, and the exps can
// start as soon as the logits are in registers.  All p >= 0, hence max p <= sum p: if both tile sums stay below 2^20
// nothing can have overflowed and the tile is committed as is.  Otherwise (first tile: reference -inf gives sum = inf;
// or a logit more than ~20 log2-units above the reference) the reference is raised to the true maximum exactly as
// Alg.1 lines 8-12 do (rescale l, acc by alpha) and the tile is evaluated again; then every p <= 1.
template <int NC>
__device__ __forceinline__ void online_update_lazy(RowState& st, const uint32_t (&r1)[NC], const uint32_t (&r2)[NC], float sc1, float sc2) {
  const float2 vsc1 = make_float2(sc1, sc1), vsc2 = make_float2(sc2, sc2);
#pragma unroll 1
  for (int attempt = 0;; ++attempt) {
    const float2 vr1 = make_float2(-st.m1, -st.m1), vr2 = make_float2(-st.m2, -st.m2);
    float2 s1v[2] = {make_float2(0.f, 0.f), make_float2(0.f, 0.f)}, s2v[2] = {s1v[0], s1v[0]}, ddv[2] = {s1v[0], s1v[0]};
#pragma unroll
    for (int e = 0; e < NC; e += 2) {
      const float2 x1 = fma2(make_float2(__uint_as_float(r1[e]), __uint_as_float(r1[e + 1])), vsc1, vr1);
      const float2 x2 = fma2(make_float2(__uint_as_float(r2[e]), __uint_as_float(r2[e + 1])), vsc2, vr2);
      const bool poly = STREAMKL_FWD_POLY_EVERY > 0 && ((e >> 1) % (STREAMKL_FWD_POLY_EVERY > 0 ? STREAMKL_FWD_POLY_EVERY : 1)) == 0;
      const float2 p1 = poly ? ex2_poly2(x1) : make_float2(ex2_approx(x1.x), ex2_approx(x1.y));
      const float2 p2 = poly ? ex2_poly2(x2) : make_float2(ex2_approx(x2.x), ex2_approx(x2.y));
      const int a = (e >> 1) & 1;
      s1v[a] = add2(s1v[a], p1);
      s2v[a] = add2(s2v[a], p2);
      ddv[a] = fma2(p1, sub2(x1, x2), ddv[a]);
    }
    const float sum1 = (s1v[0].x + s1v[0].y) + (s1v[1].x + s1v[1].y);
    const float sum2 = (s2v[0].x + s2v[0].y) + (s2v[1].x + s2v[1].y);
    const float dsum = (ddv[0].x + ddv[0].y) + (ddv[1].x + ddv[1].y);
    if ((sum1 <= 1048576.f && sum2 <= 1048576.f) || attempt >= 1) {   // (false for inf / NaN sums on the first attempt)
      st.l1 += sum1;                                                   // line 11 with alpha = 1
      st.l2 += sum2;
      st.acc += fmaf(st.m1 - st.m2, sum1, dsum);                       // line 12: sum p1 (s1' - s2')
      return;
    }
    float mx1a = -CUDART_INF_F, mx1b = -CUDART_INF_F, mx2a = -CUDART_INF_F, mx2b = -CUDART_INF_F;
#pragma unroll
    for (int e = 0; e < NC; e += 4) {
      mx1a = max3(mx1a, __uint_as_float(r1[e]), __uint_as_float(r1[e + 1]));
      mx1b = max3(mx1b, __uint_as_float(r1[e + 2]), __uint_as_float(r1[e + 3]));
      mx2a = max3(mx2a, __uint_as_float(r2[e]), __uint_as_float(r2[e + 1]));
      mx2b = max3(mx2b, __uint_as_float(r2[e + 2]), __uint_as_float(r2[e + 3]));
    }
    const float m1n = fmaxf(st.m1, fmaxf(mx1a, mx1b) * sc1), m2n = fmaxf(st.m2, fmaxf(mx2a, mx2b) * sc2);   // finite: the tile is unmasked
    const float a1 = ex2_approx(st.m1 - m1n), a2 = ex2_approx(st.m2 - m2n);                                // m = -inf gives 0
    st.l1 *= a1; st.acc *= a1; st.l2 *= a2;
    st.m1 = m1n; st.m2 = m2n;
  }
}

template <int D1, int D2, bool CAUSAL, bool SPLIT = false>
__global__ void __launch_bounds__(FwdCfg<D1, D2>::THREADS, 1)
streamkl_fwd_sm100_kernel(const __grid_constant__ CUtensorMap tmQ1, const __grid_constant__ CUtensorMap tmK1,
                          const __grid_constant__ CUtensorMap tmQ2, const __grid_constant__ CUtensorMap tmK2, const FwdParams p) {
  using C = FwdCfg<D1, D2>;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t* sQ1 = smem;
  uint8_t* sQ2 = sQ1 + C::NMT * C::KB1 * C::QBLK;
  uint8_t* sK = smem + C::Q_BYTES;
  uint64_t* bars = reinterpret_cast<uint64_t*>(sK + C::NSTAGE * C::STAGE_BYTES);
  uint64_t* q_full = bars;                    // 1
  uint64_t* k_full = bars + 1;                // NSTAGE
  uint64_t* k_empty = k_full + C::NSTAGE;     // NSTAGE
  uint64_t* s_full = k_empty + C::NSTAGE;     // [mt][st] 4
  uint64_t* s_empty = s_full + 4;             // [mt][st] 4
  uint32_t* tmem_ptr = reinterpret_cast<uint32_t*>(s_empty + 4);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  // heavy (late, causal) query tiles first within each head; consecutive CTAs share a head (K stays in L2)
  const int tile = SPLIT ? int(blockIdx.x) / p.W : int(blockIdx.x);
  const int wk = SPLIT ? int(blockIdx.x) % p.W : 0;          // key chunk of this CTA (split-K grid (b, i, w))
  const int bh = tile / p.TQ;
  const int qt = p.TQ - 1 - (tile % p.TQ);
  const int q0 = qt * C::BQ;
  const int off = p.NK - p.NQ;
  const int TK = (p.NK + C::BK - 1) / C::BK;
  const int j_begin = SPLIT ? wk * p.chunk_steps : 0;        // this CTA's 64-key steps are [j_begin, j_begin + nsteps_mt)
  const int j_end = SPLIT ? min(TK, j_begin + p.chunk_steps) : TK;

  int nsteps_mt[2] = {0, 0};
#pragma unroll
  for (int mt = 0; mt < C::NMT; ++mt) {
    const int r0 = q0 + mt * C::BM;
    int n = j_end;
    if (CAUSAL) {
      const int lastkey = min(p.NK - 1, r0 + C::BM - 1 + off);
      n = min(j_end, lastkey / C::BK + 1);
    }
    nsteps_mt[mt] = (r0 < p.NQ) ? max(0, n - j_begin) : 0;
  }
  const int nsteps = max(nsteps_mt[0], nsteps_mt[1]);

  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tmQ1); tma_prefetch_desc(&tmK1); tma_prefetch_desc(&tmQ2); tma_prefetch_desc(&tmK2);
  }
  if (warp == 1 && lane == 0) {
    mbar_init(q_full, 1);
    for (int s = 0; s < C::NSTAGE; ++s) { mbar_init(&k_full[s], 1); mbar_init(&k_empty[s], 1); }
    for (int i = 0; i < 4; ++i) { mbar_init(&s_full[i], 1); mbar_init(&s_empty[i], 4 * C::NHALF); }
    fence_mbar_init();
  }
  if (warp == 2) tmem_alloc<C::TMEM_COLS>(tmem_ptr);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_ptr;

  if (warp < 4) {
   reg_dealloc<24>();   // (pool: (96-24)*128 = 9216 >= (112-96)*512) producer / MMA / allocator warpgroup gives its registers to the two softmax warpgroups
   if (warp == 0) {
    // ===================== TMA producer =====================
    if (lane == 0) {
      const uint64_t pol_q = l2_policy_evict_first(), pol_k = l2_policy_evict_last();
      mbar_arrive_expect_tx(q_full, C::Q_BYTES);
#pragma unroll
      for (int mt = 0; mt < C::NMT; ++mt) {
#pragma unroll
        for (int kb = 0; kb < C::KB1; ++kb)
          tma_load_3d_hint(sQ1 + (mt * C::KB1 + kb) * C::QBLK, &tmQ1, q_full, kb * 64, q0 + mt * C::BM, bh, pol_q);
#pragma unroll
        for (int kb = 0; kb < C::KB2; ++kb)
          tma_load_3d_hint(sQ2 + (mt * C::KB2 + kb) * C::QBLK, &tmQ2, q_full, kb * 64, q0 + mt * C::BM, bh, pol_q);
      }
      for (int j = 0; j < nsteps; ++j) {
        const int s = j % C::NSTAGE;
        const uint32_t ph = (j / C::NSTAGE) & 1;
        mbar_wait(&k_empty[s], ph ^ 1);
        mbar_arrive_expect_tx(&k_full[s], C::STAGE_BYTES);
        uint8_t* st = sK + s * C::STAGE_BYTES;
#pragma unroll
        for (int kb = 0; kb < C::KB1; ++kb)
          tma_load_3d_hint(st + kb * C::KBLK, &tmK1, &k_full[s], kb * 64, (j_begin + j) * C::BK, bh, pol_k);
#pragma unroll
        for (int kb = 0; kb < C::KB2; ++kb)
          tma_load_3d_hint(st + (C::KB1 + kb) * C::KBLK, &tmK2, &k_full[s], kb * 64, (j_begin + j) * C::BK, bh, pol_k);
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer =====================
    // The whole warp runs the loop (warp-uniform control flow and descriptors stay in uniform registers); only the
    // tcgen05.mma / tcgen05.commit instructions themselves are issued by one elected lane.
    constexpr uint32_t idesc = umma_idesc_bf16(C::BM, C::BK, 0, 0);
    const uint64_t dq1 = umma_smem_desc_sw128(smem_u32(sQ1), 16, 1024);
    const uint64_t dq2 = umma_smem_desc_sw128(smem_u32(sQ2), 16, 1024);
    const uint64_t dk = umma_smem_desc_sw128(smem_u32(sK), 16, 1024);
    mbar_wait(q_full, 0);
    tc_fence_after();
    for (int j = 0; j < nsteps; ++j) {
      const int s = j % C::NSTAGE;
      const uint32_t ph = (j / C::NSTAGE) & 1;
      mbar_wait(&k_full[s], ph);
      tc_fence_after();
      const uint64_t dks = dk + uint64_t((s * C::STAGE_BYTES) >> 4);
      const int st = j & 1;
      const uint32_t sph = (j >> 1) & 1;
#pragma unroll
      for (int mt = 0; mt < C::NMT; ++mt) {
        if (j < nsteps_mt[mt]) {
          mbar_wait(&s_empty[mt * 2 + st], sph ^ 1);
          tc_fence_after();
          const uint32_t dS1 = tmem_base + (mt * 2 + st) * (2 * C::BK);
          const uint32_t dS2 = dS1 + C::BK;
          // Per-step descriptor bases, laundered through an empty asm so that the sixteen A descriptors are formed
          // as base + immediate next to each MMA instead of being hoisted out of the loop (32 loop-invariant 64-bit
          // values would not fit this warp's register budget: ptxas spilled them and the issue loop, not the tensor
          // pipe, set the pace of the kernel).
          uint64_t a1 = dq1 + uint64_t((mt * C::KB1 * C::QBLK) >> 4), a2 = dq2 + uint64_t((mt * C::KB2 * C::QBLK) >> 4), bk = dks;
          asm volatile("" : "+l"(a1), "+l"(a2), "+l"(bk));
          if (elect_one()) {
#pragma unroll
            for (int kb = 0; kb < C::KB1; ++kb)
#pragma unroll
              for (int k = 0; k < 4; ++k)
                umma_bf16_ss(dS1, a1 + uint64_t((kb * C::QBLK + k * 32) >> 4), bk + uint64_t((kb * C::KBLK + k * 32) >> 4), idesc,
                             (kb | k) != 0);
#pragma unroll
            for (int kb = 0; kb < C::KB2; ++kb)
#pragma unroll
              for (int k = 0; k < 4; ++k)
                umma_bf16_ss(dS2, a2 + uint64_t((kb * C::QBLK + k * 32) >> 4),
                             bk + uint64_t(((C::KB1 + kb) * C::KBLK + k * 32) >> 4), idesc, (kb | k) != 0);
            umma_commit(&s_full[mt * 2 + st]);
          }
          __syncwarp();
        }
      }
      if (elect_one()) umma_commit(&k_empty[s]);  // K stage reusable once every MMA that read it has retired
      __syncwarp();
    }
   }
  } else {
    // ===================== softmax warps =====================
    reg_alloc<112>();    // needs 16*512 = 8192 registers from the pool the other warpgroup released
    const int sw = warp - 4;
    const int quarter = warp & 3;          // TMEM lane quarter this warp may access
    const int mt = (sw >> 2) % C::NMT;
    const int half = (sw >> 2) / C::NMT;   // which 32-column group of every key tile (0 .. NHALF-1)
    const int rloc = quarter * 32 + lane;
    const int row = q0 + mt * C::BM + rloc;
    const int limit = CAUSAL ? min(p.NK - 1, row + off) : p.NK - 1;  // last visible key of this row
    const int first_row_limit = (q0 + mt * C::BM) + off;             // causal frontier of the tile's first row
    RowState st{-CUDART_INF_F, -CUDART_INF_F, 0.f, 0.f, 0.f};
    const int n = nsteps_mt[mt];
    for (int j = 0; j < n; ++j) {
      const int sg = j & 1;
      const uint32_t sph = (j >> 1) & 1;
      mbar_wait(&s_full[mt * 2 + sg], sph);
      tc_fence_after();
      const uint32_t taddr = tmem_base + (uint32_t(quarter * 32) << 16) + (mt * 2 + sg) * (2 * C::BK) + half * C::BC;
      uint32_t r1[C::BC], r2[C::BC];
      tmem_ld32(taddr, r1);
      tmem_ld32(taddr + C::BK, r2);
      tmem_wait_ld();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&s_empty[mt * 2 + sg]);  // logits are in registers: MMA may refill this stage
      const int kbase = (j_begin + j) * C::BK + half * C::BC;
      const bool masked = (CAUSAL && (kbase + C::BC - 1 > first_row_limit)) || (kbase + C::BC > p.NK);
      if (masked) online_update<true, C::BC>(st, r1, r2, p.sc1, p.sc2, kbase, limit);
#if STREAMKL_FWD_LAZY_MAX
      else        online_update_lazy<C::BC>(st, r1, r2, p.sc1, p.sc2);
#else
      else        online_update<false, C::BC>(st, r1, r2, p.sc1, p.sc2, kbase, limit);
#endif
    }
    if (n > 0) {
      // merge the column groups of each row (Eq.11 with (m2,l2) carried too, R11).  The exchange buffer aliases this
      // M-tile's own Q1 block: every MMA that reads it has completed (the last s_full of this M-tile has been observed).
      float* xch = reinterpret_cast<float*>(sQ1 + mt * C::KB1 * C::QBLK);
      if (half > 0) {
        float* x = xch + (half - 1) * 5 * C::BM;
        x[0 * C::BM + rloc] = st.m1; x[1 * C::BM + rloc] = st.l1; x[2 * C::BM + rloc] = st.m2;
        x[3 * C::BM + rloc] = st.l2; x[4 * C::BM + rloc] = st.acc;
      }
      asm volatile("bar.sync %0, %1;" ::"r"(1 + mt), "n"(C::NHALF * 128) : "memory");
      if (half == 0 && row < p.NQ) {
#pragma unroll
        for (int hb = 1; hb < C::NHALF - 1; ++hb) {   // fold groups 1 .. NHALF-2 into this thread's state; the last one below
          const float* x = xch + (hb - 1) * 5 * C::BM;
          const float m1b = x[0 * C::BM + rloc], l1b = x[1 * C::BM + rloc], m2b = x[2 * C::BM + rloc];
          const float l2b = x[3 * C::BM + rloc], accb = x[4 * C::BM + rloc];
          const float m1 = fmaxf(st.m1, m1b), m2 = fmaxf(st.m2, m2b);
          const float r1 = (m1 == -CUDART_INF_F) ? 0.f : m1, r2 = (m2 == -CUDART_INF_F) ? 0.f : m2;
          const float wa1 = exp2f(st.m1 - r1), wb1 = exp2f(m1b - r1), wa2 = exp2f(st.m2 - r2), wb2 = exp2f(m2b - r2);
          st.l1 = st.l1 * wa1 + l1b * wb1; st.l2 = st.l2 * wa2 + l2b * wb2; st.acc = st.acc * wa1 + accb * wb1;
          st.m1 = m1; st.m2 = m2;
        }
        const float* xl = xch + (C::NHALF - 2) * 5 * C::BM;
        const float m1b = xl[0 * C::BM + rloc], l1b = xl[1 * C::BM + rloc], m2b = xl[2 * C::BM + rloc];
        const float l2b = xl[3 * C::BM + rloc], accb = xl[4 * C::BM + rloc];
        const float m1 = fmaxf(st.m1, m1b), m2 = fmaxf(st.m2, m2b);
        // unsplit: half 0 holds key 0, so the maxima are finite.  A split-K chunk can lie wholly past a row's causal
        // frontier: both halves are then (-inf, 0, 0) and the reference is 0 (R7), giving the identity partial.
        const float r1 = (SPLIT && m1 == -CUDART_INF_F) ? 0.f : m1, r2 = (SPLIT && m2 == -CUDART_INF_F) ? 0.f : m2;
        const float wa1 = exp2f(st.m1 - r1), wb1 = exp2f(m1b - r1), wa2 = exp2f(st.m2 - r2), wb2 = exp2f(m2b - r2);
        const float l1 = st.l1 * wa1 + l1b * wb1, l2 = st.l2 * wa2 + l2b * wb2, acc = st.acc * wa1 + accb * wb1;
        if constexpr (SPLIT) {   // partial statistics of this key chunk (log2 domain), merged by the reduce kernel
          float* o = p.part + (size_t(bh) * p.W + wk) * 5 * size_t(p.NQ) + row;
          o[0] = m1; o[size_t(p.NQ)] = l1; o[2 * size_t(p.NQ)] = m2; o[3 * size_t(p.NQ)] = l2; o[4 * size_t(p.NQ)] = acc;
        } else {
        // Alg.1 lines 13-15 in natural-log units (R6): LSE = ln2*(m + log2 l); KL = ln2*acc/l1 + LSE2 - LSE1
        const float LN2 = 0.6931471805599453f;
        const float e1 = LN2 * (m1 + log2f(l1));
        const float e2 = LN2 * (m2 + log2f(l2));
        const size_t o = size_t(bh) * p.NQ + row;
        p.lse1[o] = e1;
        p.lse2[o] = e2;
        p.kl[o] = fmaf(LN2, acc / l1, e2 - e1);
        }
      }
    } else if (SPLIT && half == 0 && row < p.NQ) {   // no step of this chunk is visible to this M-tile: identity partial
      float* o = p.part + (size_t(bh) * p.W + wk) * 5 * size_t(p.NQ) + row;
      o[0] = -CUDART_INF_F; o[size_t(p.NQ)] = 0.f; o[2 * size_t(p.NQ)] = -CUDART_INF_F; o[3 * size_t(p.NQ)] = 0.f;
      o[4 * size_t(p.NQ)] = 0.f;
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 2) {
    tc_fence_after();
    tmem_dealloc<C::TMEM_COLS>(tmem_base);
  }
}

// Split-K reduce (Eq.11; (m2,l2) merged the same way, R11): one thread per query row folds the W
// partials in chunk order and finishes Alg.1 lines 13-15.  Chunk 0 always sees key 0, so the merged maxima are finite.
__global__ void streamkl_fwd_splitk_reduce_kernel(const float* __restrict__ part, int NQ, int W, long long total_rows,
                                                  float* __restrict__ kl, float* __restrict__ lse1, float* __restrict__ lse2) {
  const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= total_rows) return;
  const long long bh = idx / NQ;
  const int row = int(idx % NQ);
  const float* b = part + size_t(bh) * W * 5 * size_t(NQ) + row;
  float m1 = b[0], l1 = b[size_t(NQ)], m2 = b[2 * size_t(NQ)], l2 = b[3 * size_t(NQ)], acc = b[4 * size_t(NQ)];
  for (int w = 1; w < W; ++w) {
    const float* c = b + size_t(w) * 5 * size_t(NQ);
    const float m1b = c[0], l1b = c[size_t(NQ)], m2b = c[2 * size_t(NQ)], l2b = c[3 * size_t(NQ)], accb = c[4 * size_t(NQ)];
    const float n1 = fmaxf(m1, m1b), n2 = fmaxf(m2, m2b);
    const float wa1 = exp2f(m1 - n1), wb1 = exp2f(m1b - n1), wa2 = exp2f(m2 - n2), wb2 = exp2f(m2b - n2);
    l1 = l1 * wa1 + l1b * wb1; acc = acc * wa1 + accb * wb1; l2 = l2 * wa2 + l2b * wb2;
    m1 = n1; m2 = n2;
  }
  const float LN2 = 0.6931471805599453f;
  const float e1 = LN2 * (m1 + log2f(l1)), e2 = LN2 * (m2 + log2f(l2));
  lse1[idx] = e1;
  lse2[idx] = e2;
  kl[idx] = fmaf(LN2, acc / l1, e2 - e1);
}

}  // namespace skl
