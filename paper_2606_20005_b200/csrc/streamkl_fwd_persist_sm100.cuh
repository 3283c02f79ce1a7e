// streamkl_fwd_persist_sm100.cuh -- the fixed-plan forward kernel (streamkl_fwd_sm100.cuh, Algorithm 1) as a
// PERSISTENT kernel: one CTA per SM loops over (head, Q tile) work items instead of one CTA per item.
//
// Why.  With one CTA per SM (512 TMEM columns, ~200 KB of shared memory) nothing overlaps a tile's prologue (TMEM allocation,
// barrier initialisation, the Q load from HBM, the first logit MMAs) and epilogue (Eq.11 merge, stores, CTA exit, next CTA's
// launch): ncu on cfg 3 (16K keys, 64.5 steps per tile on average) shows 2153 cycles per step over the kernel against 1926 inside
// the step loop -- 10.5 % of the time is spent between tiles (cfg 4, 258 steps per tile: 2.6 %).  Here TMEM and the barriers are
// set up once; the producer fetches the next item (dynamic: an atomic counter, so the causal imbalance is absorbed as the
// hardware block scheduler absorbed it), waits only for the MMAs of the previous tile to release the Q buffer, and loads the
// next Q and K stages while the softmax warps are still working on the previous tile's last two steps; the issuer starts the
// next tile's logits as soon as a TMEM stage is free.
//
// Work order = the non-persistent kernel's block order (heads consecutive, heavy causal tiles first within a head), so the K
// tiles of the few heads in flight stay in L2.  Per-row arithmetic is unchanged: results are bit-identical.
#pragma once
#include "streamkl_fwd_sm100.cuh"

namespace skl {

template <int D1, int D2>
struct FwdPersistCfg : FwdCfg<D1, D2> {
  using B = FwdCfg<D1, D2>;
  static constexpr int XCH_BYTES = 2 * (B::NGRP - 1) * 5 * B::BM * 4;   // two Eq.11 exchange buffers (alternating per tile)
  static constexpr int AUX_BYTES = 512;
  static constexpr int NSTAGE_RAW = (B::SMEM_LIMIT - 1024 - AUX_BYTES - XCH_BYTES - B::Q_BYTES) / B::STAGE_BYTES;
  static constexpr int NSTAGE = NSTAGE_RAW > 6 ? 6 : NSTAGE_RAW;
  static_assert(NSTAGE >= 2, "need at least a double-buffered K ring");
  static constexpr int SMEM_BYTES = 1024 + B::Q_BYTES + NSTAGE * B::STAGE_BYTES + XCH_BYTES + AUX_BYTES;
};

// sched[0] = next work item beyond the first wave, sched[1] = CTAs that have finished; both 0 between launches
template <int D1, int D2, bool CAUSAL>
__global__ void __launch_bounds__(FwdCfg<D1, D2>::THREADS, 1)
streamkl_fwd_persist_sm100_kernel(const __grid_constant__ CUtensorMap tmQ1, const __grid_constant__ CUtensorMap tmK1,
                                  const __grid_constant__ CUtensorMap tmQ2, const __grid_constant__ CUtensorMap tmK2, const FwdParams p,
                                  int* __restrict__ sched) {
  using C = FwdPersistCfg<D1, D2>;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t* sQ1 = smem;
  uint8_t* sQ2 = sQ1 + C::KB1 * C::QBLK;
  uint8_t* sK = smem + C::Q_BYTES;
  float* sXch = reinterpret_cast<float*>(sK + C::NSTAGE * C::STAGE_BYTES);
  uint64_t* bars = reinterpret_cast<uint64_t*>(reinterpret_cast<uint8_t*>(sXch) + C::XCH_BYTES);
  uint64_t* q_full = bars;                    // 1  Q tile of the current item landed
  uint64_t* q_empty = bars + 1;               // 1  every MMA of the item has retired: the Q buffer may be overwritten
  uint64_t* k_full = bars + 2;                // NSTAGE
  uint64_t* k_empty = k_full + C::NSTAGE;     // NSTAGE
  uint64_t* s_full = k_empty + C::NSTAGE;     // 2
  uint64_t* s_empty = s_full + 2;             // 2
  uint64_t* t_full = s_empty + 2;             // 2  work-item ring: written by the producer
  uint64_t* t_empty = t_full + 2;             // 2  read by the issuer warp and the sixteen softmax warps
  int* t_ring = reinterpret_cast<int*>(t_empty + 2);     // 2 work items (-1 = no more work)
  uint32_t* tmem_ptr = reinterpret_cast<uint32_t*>(t_ring + 2);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int total = p.TQ * p.BH;
  const int off = p.NK - p.NQ;
  const int TK = (p.NK + C::BK - 1) / C::BK;
  // work item -> (head, Q tile): the block order of the non-persistent kernel
  auto item_q0 = [&](int item) { return (p.TQ - 1 - (item % p.TQ)) * C::BQ; };
  auto item_steps = [&](int q0) { return CAUSAL ? min(TK, min(p.NK - 1, q0 + C::BM - 1 + off) / C::BK + 1) : TK; };

  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tmQ1); tma_prefetch_desc(&tmK1); tma_prefetch_desc(&tmQ2); tma_prefetch_desc(&tmK2);
  }
  if (warp == 1 && lane == 0) {
    mbar_init(q_full, 1);
    mbar_init(q_empty, 1);
    for (int s = 0; s < C::NSTAGE; ++s) { mbar_init(&k_full[s], 1); mbar_init(&k_empty[s], 1); }
    for (int i = 0; i < 2; ++i) {
      mbar_init(&s_full[i], 1); mbar_init(&s_empty[i], 4 * C::NGRP);
      mbar_init(&t_full[i], 1); mbar_init(&t_empty[i], 1 + 4 * C::NGRP);
    }
    fence_mbar_init();
  }
  if (warp == 2) tmem_alloc<C::TMEM_COLS>(tmem_ptr);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_ptr;

  // every consumer warp takes the next work item from the ring (warp-uniform); -1 ends the loop
  auto next_item = [&](int n) {
    const int ts = n & 1;
    mbar_wait(&t_full[ts], (n >> 1) & 1);
    const int item = *reinterpret_cast<volatile int*>(&t_ring[ts]);
    __syncwarp();
    if (lane == 0) mbar_arrive(&t_empty[ts]);
    return item;
  };

  if (warp < 4) {
   reg_dealloc<32>();   // (128 * (96 - 32) = 8192 registers = what the sixteen softmax warps take: 512 * (112 - 96))
   if (warp == 0) {
    // ===================== scheduler + TMA producer =====================
    if (lane == 0) {
      const uint64_t pol_q = l2_policy_evict_first(), pol_k = l2_policy_evict_last();
      int kc = 0;                                   // K stages issued so far (ring position persists across items)
      int item = int(blockIdx.x);                   // first wave: static; afterwards the shared counter
      for (int n = 0;; ++n) {
        const int ts = n & 1;
        mbar_wait(&t_empty[ts], ((n >> 1) & 1) ^ 1);
        t_ring[ts] = item < total ? item : -1;
        mbar_arrive(&t_full[ts]);                   // (release: the ring entry is visible to whoever observes the phase)
        if (item >= total) break;
        const int bh = item / p.TQ;
        const int hq = bh % p.H, bq = bh / p.H, hk = hq / p.G;
        const int q0 = item_q0(item);
        const int nsteps = item_steps(q0);
        mbar_wait(q_empty, (n & 1) ^ 1);            // the previous item's MMAs have retired (passes at once for the first item)
        mbar_arrive_expect_tx(q_full, C::Q_BYTES);
#pragma unroll
        for (int kb = 0; kb < C::KB1; ++kb) tma_load_4d_hint(sQ1 + kb * C::QBLK, &tmQ1, q_full, kb * 64, q0, hq, bq, pol_q);
#pragma unroll
        for (int kb = 0; kb < C::KB2; ++kb) tma_load_4d_hint(sQ2 + kb * C::QBLK, &tmQ2, q_full, kb * 64, q0, hq, bq, pol_q);
        for (int j = 0; j < nsteps; ++j, ++kc) {
          const int s = kc % C::NSTAGE;
          mbar_wait(&k_empty[s], ((kc / C::NSTAGE) & 1) ^ 1);
          mbar_arrive_expect_tx(&k_full[s], C::STAGE_BYTES);
          uint8_t* st = sK + s * C::STAGE_BYTES;
#pragma unroll
          for (int kb = 0; kb < C::KB1; ++kb) tma_load_4d_hint(st + kb * C::KBLK, &tmK1, &k_full[s], kb * 64, j * C::BK, hk, bq, pol_k);
#pragma unroll
          for (int kb = 0; kb < C::KB2; ++kb)
            tma_load_4d_hint(st + (C::KB1 + kb) * C::KBLK, &tmK2, &k_full[s], kb * 64, j * C::BK, hk, bq, pol_k);
        }
        // take the next item only now, when this one's loads are all issued: a ticket taken earlier is an item reserved for a whole
        // tile time (measured: SM finish times 7.3-8.0 M cycles instead of 7.6-7.8 M at 32K); its latency hides behind the wait for
        // q_empty, which needs this item's last MMAs to retire anyway
        item = int(gridDim.x) + atomicAdd(&sched[0], 1);
      }
    }
   } else if (warp == 1) {
    // ===================== MMA issuer =====================
    const uint32_t idesc = umma_idesc_16(C::BM, C::BK, 0, 0, p.fmt16);
    const uint64_t dq1 = umma_smem_desc_sw128(smem_u32(sQ1), 16, 1024);
    const uint64_t dq2 = umma_smem_desc_sw128(smem_u32(sQ2), 16, 1024);
    const uint64_t dk = umma_smem_desc_sw128(smem_u32(sK), 16, 1024);
    int kc = 0, g = 0;                              // K stages / logit steps so far over all items of this CTA
    for (int n = 0;; ++n) {
      const int item = next_item(n);
      if (item < 0) break;
      const int nsteps = item_steps(item_q0(item));
      mbar_wait(q_full, n & 1);
      tc_fence_after();
      for (int j = 0; j < nsteps; ++j, ++kc, ++g) {
        const int s = kc % C::NSTAGE;
        mbar_wait(&k_full[s], (kc / C::NSTAGE) & 1);
        const int st = g & 1;
        mbar_wait(&s_empty[st], ((g >> 1) & 1) ^ 1);
        tc_fence_after();
        const uint32_t dS1 = tmem_base + st * (2 * C::BK);
        const uint32_t dS2 = dS1 + C::BK;
        uint64_t a1 = dq1, a2 = dq2, bk = dk + uint64_t((s * C::STAGE_BYTES) >> 4);
        asm volatile("" : "+l"(a1), "+l"(a2), "+l"(bk));   // descriptors = base + immediate beside each MMA (see streamkl_fwd_sm100.cuh)
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
          umma_commit(&s_full[st]);
          umma_commit(&k_empty[s]);
          if (j + 1 == nsteps) umma_commit(q_empty);   // the item's last MMAs: the Q buffer is free once they retire
        }
        __syncwarp();
      }
      if (nsteps & 1) {
        // an item with an odd number of steps is padded by one EMPTY step, so that every item starts on TMEM stage 0 and the
        // softmax loop keeps compile-time stage addresses: take the stage, hand it over at once (no MMA), the softmax warps release it
        const int st = g & 1;
        mbar_wait(&s_empty[st], ((g >> 1) & 1) ^ 1);
        if (elect_one()) umma_commit(&s_full[st]);
        __syncwarp();
        ++g;
      }
    }
   }
  } else {
    // ===================== softmax warps =====================
    reg_alloc<112>();
    const int quarter = warp & 3;
    const int grp = (warp - 4) >> 2;
    const int rloc = quarter * 32 + lane;
    const float sc1 = p.sc1, sc2 = p.sc2;
    const uint32_t tbase = tmem_base + (uint32_t(quarter * 32) << 16) + grp * C::BC;
    const bool relu2 = p.act2 == 1;
    int g0 = 0;                                     // logit steps of the earlier items of this CTA: step j of an item is global step g0 + j
    for (int n = 0;; ++n) {
      const int item = next_item(n);
      if (item < 0) break;
      const int bh = item / p.TQ;
      const int q0 = item_q0(item);
      const int nsteps = item_steps(q0);
      const int row = q0 + rloc;
      const int limit = CAUSAL ? min(p.NK - 1, row + off) : p.NK - 1;
      const int vis_all = CAUSAL ? min(p.NK - 1, q0 + off) : p.NK - 1;
      const int kg = vis_all - (C::BC - 1) - grp * C::BC;
      const int n_fast = kg < 0 ? 0 : max(0, min(nsteps, kg / C::BK + 1));
      RowState st{-CUDART_INF_F, -CUDART_INF_F, make_float2(0.f, 0.f), make_float2(0.f, 0.f), make_float2(0.f, 0.f)};
      // TMEM stage / barrier / phase of step j of this item (g0 is even: items are padded to an even number of steps)
      auto stage_addr = [&](int j) { return tbase + uint32_t(j & 1) * (2 * C::BK); };
      auto full_bar = [&](int j) { return &s_full[j & 1]; };
      auto empty_bar = [&](int j) { return &s_empty[j & 1]; };
      auto full_par = [&](int j) { return uint32_t((g0 + j) >> 1) & 1u; };
      auto wait_full = [&](int j) {
        mbar_wait(full_bar(j), full_par(j));
        tc_fence_after();
      };
      auto release = [&](uint64_t* bar) {
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(bar);
      };

      auto run_fast = [&](auto relu_tag) {
        constexpr bool RELU2 = decltype(relu_tag)::value;
        LogitChunk A;
        XChunk X;
        wait_full(0);
        ld_chunk(stage_addr(0), A);
        wait_chunk(A);
        {
          float mx1 = __uint_as_float(A.a[0]), mx2 = __uint_as_float(A.b[0]);
#pragma unroll
          for (int e = 1; e < 8; e += 2) {
            mx1 = max3(mx1, __uint_as_float(A.a[e]), __uint_as_float(A.a[(e + 1) & 7]));
            mx2 = max3(mx2, __uint_as_float(A.b[e]), __uint_as_float(A.b[(e + 1) & 7]));
          }
          st.m1 = mx1 * sc1;
          st.m2 = RELU2 ? fmaxf(mx2 * sc2, 0.f) : mx2 * sc2;
        }
        float nm1 = -st.m1, nm2 = -st.m2;
        // one step: identical to fast_step of streamkl_fwd_sm100.cuh (see the comments there)
        auto fast_step = [&](auto masked_tag, const uint32_t tcur, const uint32_t tnext, uint64_t* full_next, const uint32_t par_next,
                             uint64_t* empty_cur, const bool has_next, const int k0) {
          constexpr bool MASKED = decltype(masked_tag)::value;
          constexpr uint32_t PMASK = MASKED ? 0u : C::POLY_MASK;
          float2 T1, T2, TD;
          wait_chunk(A);
          scale_chunk<RELU2, MASKED>(A, sc1, sc2, nm1, nm2, X, k0, limit);
          ld_chunk(tcur + 8, A);
          pin_below(X);
          accumulate_chunk<(PMASK >> 0) & 15u, true>(X, T1, T2, TD);
          wait_chunk(A);
          scale_chunk<RELU2, MASKED>(A, sc1, sc2, nm1, nm2, X, k0 + 8, limit);
          ld_chunk(tcur + 16, A);
          pin_below(X);
          accumulate_chunk<(PMASK >> 4) & 15u, false>(X, T1, T2, TD);
          wait_chunk(A);
          scale_chunk<RELU2, MASKED>(A, sc1, sc2, nm1, nm2, X, k0 + 16, limit);
          ld_chunk(tcur + 24, A);
          const bool ready = has_next && mbar_test_wait(full_next, par_next);
          pin_below(X);
          accumulate_chunk<(PMASK >> 8) & 15u, false>(X, T1, T2, TD);
          wait_chunk(A);
          scale_chunk<RELU2, MASKED>(A, sc1, sc2, nm1, nm2, X, k0 + 24, limit);
          if (has_next) {
            if (!ready) mbar_wait(full_next, par_next);
            tc_fence_after();
            ld_chunk(tnext, A);
          }
          pin_below(X);
          accumulate_chunk<(PMASK >> 12) & 15u, false>(X, T1, T2, TD);
          const float chk = (T1.x + T1.y) + (T2.x + T2.y);
          if (!__any_sync(0xffffffffu, !(chk <= 1048576.f))) {
            st.R1 = add2(st.R1, T1);
            st.R2 = add2(st.R2, T2);
            st.RD = add2(st.RD, TD);
          } else {
            st = MASKED ? safe_step<true>(tcur, st, sc1, sc2, k0, limit, RELU2) : safe_step<false>(tcur, st, sc1, sc2, 0, 0, RELU2);
            nm1 = -st.m1;
            nm2 = -st.m2;
          }
          release(empty_cur);
        };
        const uint32_t t0 = tbase, t1 = tbase + 2 * C::BK;
        uint32_t par = uint32_t(g0 >> 1) & 1u;   // parity of the s_full phases of the step pair (2i, 2i+1)
        int j = 0;
        for (; j + 2 <= n_fast; j += 2) {
          fast_step(std::false_type{}, t0, t1, &s_full[1], par, &s_empty[0], j + 1 < nsteps, 0);
          fast_step(std::false_type{}, t1, t0, &s_full[0], par ^ 1, &s_empty[1], j + 2 < nsteps, 0);
          par ^= 1;
        }
        for (; j < nsteps; ++j) {
          const uint32_t tc = stage_addr(j), tn = stage_addr(j + 1);
          if (j < n_fast) fast_step(std::false_type{}, tc, tn, full_bar(j + 1), full_par(j + 1), empty_bar(j), j + 1 < nsteps, 0);
          else            fast_step(std::true_type{}, tc, tn, full_bar(j + 1), full_par(j + 1), empty_bar(j), j + 1 < nsteps, j * C::BK + grp * C::BC);
        }
      };
      if (n_fast > 0) {
        if (relu2) run_fast(std::true_type{}); else run_fast(std::false_type{});
      } else {
        for (int j = 0; j < nsteps; ++j) {
          wait_full(j);
          st = safe_step<true>(stage_addr(j), st, sc1, sc2, j * C::BK + grp * C::BC, limit, relu2);
          release(empty_bar(j));
        }
      }
      if (nsteps & 1) {   // the item's padding step (see the issuer): nothing to read, hand the stage back
        wait_full(nsteps);
        release(empty_bar(nsteps));
      }
      g0 += (nsteps + 1) & ~1;

      // Eq.11 merge of the four column groups of each row (R11) and Alg.1 lines 13-15, through this item's exchange buffer
      const float pl1 = st.R1.x + st.R1.y, pl2 = st.R2.x + st.R2.y;
      const float pacc = (st.m1 == -CUDART_INF_F) ? 0.f : fmaf(st.m1 - st.m2, pl1, st.RD.x + st.RD.y);
      float* xch = sXch + (n & 1) * ((C::NGRP - 1) * 5 * C::BM);
      if (grp > 0) {
        float* x = xch + (grp - 1) * 5 * C::BM;
        x[0 * C::BM + rloc] = st.m1; x[1 * C::BM + rloc] = pl1; x[2 * C::BM + rloc] = st.m2;
        x[3 * C::BM + rloc] = pl2; x[4 * C::BM + rloc] = pacc;
      }
      asm volatile("bar.sync 1, %0;" ::"n"(C::NGRP * 128) : "memory");
      if (grp == 0 && row < p.NQ) {
        float m1 = st.m1, m2 = st.m2, l1 = pl1, l2 = pl2, acc = pacc;
#pragma unroll
        for (int hb = 1; hb < C::NGRP; ++hb) {
          const float* x = xch + (hb - 1) * 5 * C::BM;
          const float m1b = x[0 * C::BM + rloc], l1b = x[1 * C::BM + rloc], m2b = x[2 * C::BM + rloc];
          const float l2b = x[3 * C::BM + rloc], accb = x[4 * C::BM + rloc];
          const float n1 = fmaxf(m1, m1b), n2 = fmaxf(m2, m2b);
          const float r1 = (n1 == -CUDART_INF_F) ? 0.f : n1, r2 = (n2 == -CUDART_INF_F) ? 0.f : n2;
          const float wa1 = exp2f(m1 - r1), wb1 = exp2f(m1b - r1), wa2 = exp2f(m2 - r2), wb2 = exp2f(m2b - r2);
          l1 = l1 * wa1 + l1b * wb1; l2 = l2 * wa2 + l2b * wb2; acc = acc * wa1 + accb * wb1;
          m1 = n1; m2 = n2;
        }
        const float LN2 = 0.6931471805599453f;
        const float e1 = LN2 * (m1 + log2f(l1));
        const float e2 = LN2 * (m2 + log2f(l2));
        const size_t o = size_t(bh) * p.NQ + row;
        p.lse1[o] = e1;
        p.lse2[o] = e2;
        p.kl[o] = fmaf(LN2, acc / l1, e2 - e1);
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 2) {
    tc_fence_after();
    tmem_dealloc<C::TMEM_COLS>(tmem_base);
  }
  // the last CTA to finish rearms the scheduler for the next launch that uses this slot
  if (threadIdx.x == 0) {
    const int done = atomicAdd(&sched[1], 1);
    if (done == int(gridDim.x) - 1) {
      sched[0] = 0;
      sched[1] = 0;
      __threadfence();
    }
  }
}

}  // namespace skl
