// streamkl_fwd_sm100.cuh -- StreamKL forward (Algorithm 1) for sm_100a.
//
// One CTA owns one 128-row Q tile of one (b,h) and streams 128-key tiles (N=128 logit MMAs):
//   warp 0      TMA producer : Q1,Q2 once; K1_j,K2_j through an NSTAGE ring          (F1, F2 of DESIGN.md)
//   warp 1      MMA issuer   : S1 = Q1 K1_j^T, S2 = Q2 K2_j^T, tcgen05.mma -> TMEM    (F3)
//   warp 2      TMEM allocator
//   warps 4-19  sixteen softmax warps = 4 column groups (32 keys of every tile) x 4 TMEM lane quarters    (F4, F5, F6)
// TMEM (512 columns): two stages of {S1 (128 cols), S2 (128 cols)}.  A softmax thread owns ONE query row and ONE 32-column
// group of every key tile and keeps its own partial statistics over that key subset, entirely thread-locally in the log2
// domain (exp2 instead of exp; R6); the four groups of a row are merged once, after the last tile,
// with the associative merge of Eq.11 (carrying (m2,l2) too: R11).
//
// The per-thread stream (v2).  A step's 32+32 logits are pulled from TMEM in CHUNKS of 8+8 columns, the load of the next
// chunk (the next step's first chunk included) issued before the current one is evaluated, so a thread never waits for
// TMEM, holds 32 instead of 64 logit registers, and -- because ptxas cannot move a chunk's arithmetic above the
// tcgen05.wait::ld it depends on -- the MUFU exps and the FMA-pipe polynomial exps stay interleaved at chunk granularity
// instead of being sorted into one polynomial phase and one MUFU phase per step (the v1 schedule; MUFU sat idle whenever
// all four warps of a sub-partition were in their polynomial phase).
//
// Running state per thread, relative to a reference (m1, m2) that is NOT the running maximum (DESIGN.md 6.1 "lazy reference";
// Eq.8-10 hold for any reference as long as the sums are relative to it):
//     R1 = sum 2^x1,  R2 = sum 2^x2,  RD = sum 2^x1 (x1 - x2),   x_t = s_t sc_t - m_t,   kept as packed fp32x2 lane pairs;
// Alg.1's (l1, l2, acc) are l_t = R_t and acc = RD + (m1 - m2) R1 (log2 units), formed once per tile.  A step accumulates
// into step-local sums T first; since every p >= 0, sum(T1) + sum(T2) <= 2^20 proves no p exceeded 2^20 (nothing overflowed,
// the polynomial's clamp was not hit) and T is committed.  Otherwise the step is done again by `safe_step` from the logits
// still in TMEM (the stage is released only after the check): true row maximum, Alg.1 lines 8-12 (rescale by alpha), p <= 1.
// Masked steps (causal diagonal, key tails) always take `safe_step`.
#pragma once
#include <cuda_bf16.h>
#include <math_constants.h>

#include <type_traits>

#include "sm100_ptx.cuh"

// Which of the 16 column pairs a thread evaluates per step take their two exps on the FMA pipe (ex2_poly2) instead of
// MUFU: one 4-bit mask per chunk (bit u = column pair u of the chunk), chunks 0..3 in nibbles 0..3.  The forward is
// MUFU-bound 2:1 (d1 + d2 = 256) to 2.7:1 (192) against the tensor pipe, but it also runs into the 1000 W cap, and a
// polynomial exp costs six times the instructions of a MUFU one.  Measured in a sustained loop on B200:
// d = 128/128: 2/16 10.23 ms, 3/16 9.97, 4/16 10.08, 5/16 10.37 (cfg4 with 8 heads); d = 128/64: 3/16 2.355 ms, 4/16 2.343,
// 5/16 2.42, 6/16 2.47 (cfg3).
#ifndef STREAMKL_FWD_POLY_MASK_WIDE
#define STREAMKL_FWD_POLY_MASK_WIDE 0x1011u   // d1 + d2 = 256: three column pairs in sixteen
#endif
#ifndef STREAMKL_FWD_POLY_MASK_NARROW
#define STREAMKL_FWD_POLY_MASK_NARROW 0x1111u // d1 + d2 < 256: a quarter of the exps
#endif

namespace skl {

template <int D1, int D2>
struct FwdCfg {
  static_assert(D1 % 64 == 0 && D2 % 64 == 0 && D1 >= 64 && D2 >= 64 && D1 <= 128 && D2 <= 128, "fixed plans: d in {64,128}");
  static constexpr bool BLOCKED = false;     // whole {K1_j, K2_j} stages in the ring (FwdCfg<0,0>: single K-blocks)
  static constexpr int BM = 128;             // rows per Q tile (TMEM lanes)
  static constexpr int BK = 128;             // keys per step = N of the logit MMAs
  static constexpr int BQ = BM;              // query rows per CTA
  static constexpr int KB1 = D1 / 64, KB2 = D2 / 64;  // 128-byte K-blocks per row
  static constexpr int QBLK = BM * 128;      // bytes of one [128 rows x 64 bf16] swizzled block
  static constexpr int KBLK = BK * 128;
  static constexpr int Q_BYTES = (KB1 + KB2) * QBLK;
  static constexpr int STAGE_BYTES = (KB1 + KB2) * KBLK;
  static constexpr int SMEM_LIMIT = 227 * 1024;
  static constexpr int AUX_BYTES = 256;      // barriers + tmem pointer
  static constexpr int NSTAGE_RAW = (SMEM_LIMIT - 1024 - AUX_BYTES - Q_BYTES) / STAGE_BYTES;
  static constexpr int NSTAGE = NSTAGE_RAW > 6 ? 6 : NSTAGE_RAW;
  static_assert(NSTAGE >= 2, "need at least a double-buffered K ring");
  static constexpr int SMEM_BYTES = 1024 + Q_BYTES + NSTAGE * STAGE_BYTES + AUX_BYTES;
  static constexpr int NGRP = 4;             // column groups of a key tile (one softmax thread per row and group)
  static constexpr int BC = BK / NGRP;       // columns per softmax thread and step (32)
  static constexpr int CH = 8;               // columns per TMEM chunk load
  static constexpr int NCH = BC / CH;        // chunks per step (4)
  static constexpr int THREADS = 128 + NGRP * 128;
  static constexpr uint32_t TMEM_COLS = 512;
  static constexpr uint32_t POLY_MASK = (D1 + D2 == 256) ? STREAMKL_FWD_POLY_MASK_WIDE : STREAMKL_FWD_POLY_MASK_NARROW;
};

// Head dims beyond 128 (padded to 192 / 256): Q alone is up to 128 KB, so a whole 128-key stage of K1,K2 no longer fits beside
// it.  FwdCfg<0, 0> is the BLOCKED plan: the numbers of 64-element K-blocks per row (kb1, kb2) are run-time, K is streamed
// through a ring of single [128 keys x 64 elements] blocks (16 KB each, one full / empty barrier pair per block) and the issuer
// accumulates a step's logits block by block.  TMEM plan, softmax warps and epilogue are those of the fixed plans.
template <>
struct FwdCfg<0, 0> {
  static constexpr bool BLOCKED = true;
  static constexpr int BM = 128, BK = 128, BQ = BM;
  static constexpr int KB1 = 0, KB2 = 0;                 // run-time (FwdParams::kb1, kb2)
  static constexpr int QBLK = BM * 128, KBLK = BK * 128;
  static constexpr int MAX_RING = 12;
  static constexpr int AUX_BYTES = 512;
  static constexpr int SMEM_LIMIT = 227 * 1024;
  static constexpr int Q_BYTES = 0, STAGE_BYTES = KBLK, NSTAGE = MAX_RING;   // (unused by the blocked branches)
  static constexpr int NGRP = 4, BC = BK / NGRP, CH = 8, NCH = BC / CH;
  static constexpr int THREADS = 128 + NGRP * 128;
  static constexpr uint32_t TMEM_COLS = 512;
  static constexpr uint32_t POLY_MASK = STREAMKL_FWD_POLY_MASK_WIDE;
  // ring blocks that fit beside the resident Q tile (host side)
  // (`slot` = bytes of a ring entry: a whole K-block, or this CTA's half of it under the cta_group::2 plan, whose ring may have 16 entries)
  static constexpr int ring_blocks(int kb1, int kb2, int slot = KBLK) {
    const int r = (SMEM_LIMIT - 1024 - AUX_BYTES - (kb1 + kb2) * QBLK) / slot;
    const int cap = slot == KBLK ? MAX_RING : 16;
    return r > cap ? cap : r;
  }
  static constexpr int smem_bytes(int kb1, int kb2, int slot = KBLK) {
    return 1024 + (kb1 + kb2) * QBLK + ring_blocks(kb1, kb2, slot) * slot + AUX_BYTES;
  }
};

struct FwdParams {
  int NQ, NK, TQ;       // TQ = number of 128-row Q tiles per head
  int kb1, kb2, nring;  // BLOCKED plan only: 64-element K-blocks per row of distribution 1 / 2, ring size in blocks
  int BH;               // B * H query heads
  int H, G;             // query heads per batch; query heads per K head (GQA: query head h reads K head h / G)
  uint32_t fmt16;       // operand format of the logit MMAs: 1 bf16, 0 fp16
  int act2;             // student activation: 0 none, 1 relu -- s2 = relu(c2 <q2,k2>) before its softmax (R23)
  float sc1, sc2;       // c_t * log2(e)
  float* kl;
  float* lse1;
  float* lse2;
  // split-K: W contiguous key chunks of `chunk_steps` 128-key steps each; partial statistics
  // (m1,l1,m2,l2,acc in the log2 domain) go to part[bh][w][5][NQ] and streamkl_fwd_splitk_reduce_kernel merges them
  int W, chunk_steps;
  float* part;
};

// Per-thread running state (see the header comment).  m = -inf means "no visible key yet" (then R = 0).
struct RowState {
  float m1, m2;
  float2 R1, R2, RD;
};

// TMEM -> registers: 8 columns of S1 and the matching 8 columns of S2 (128 TMEM columns further) for this warp's 32 lanes
struct LogitChunk {
  uint32_t a[8], b[8];
};
__device__ __forceinline__ void ld_chunk(uint32_t taddr, LogitChunk& c) {
  tmem_ld8(taddr, c.a);
  tmem_ld8(taddr + 128, c.b);
}
// tcgen05.wait::ld with the chunk's registers tied in, so that the compiler keeps every use of them after the wait
__device__ __forceinline__ void wait_chunk(LogitChunk& c) {
  asm volatile("tcgen05.wait::ld.sync.aligned;"
               : "+r"(c.a[0]), "+r"(c.a[1]), "+r"(c.a[2]), "+r"(c.a[3]), "+r"(c.a[4]), "+r"(c.a[5]), "+r"(c.a[6]), "+r"(c.a[7]),
                 "+r"(c.b[0]), "+r"(c.b[1]), "+r"(c.b[2]), "+r"(c.b[3]), "+r"(c.b[4]), "+r"(c.b[5]), "+r"(c.b[6]), "+r"(c.b[7])
               :: "memory");
}

// A chunk's logits as shifted log2-domain exponents x_t = s_t sc_t - m_t, 4 column pairs per distribution (packed fp32x2).
// Forming them is the ONLY read of the raw logit registers, so the next tcgen05.ld may target the same registers at once.
struct XChunk {
  float2 x1[4], x2[4];
};
// RELU2: the student's logit is relu(s2 sc2) (R23): relu(y) - m = max(y - m, -m).
// MASKED (causal diagonal tiles, key tails): a key beyond `limit` gets x1 = x2 = kMaskedX, so that both of its P~ are exactly 0
// (ex2.approx.ftz of a hugely negative argument) and its S1 - S2 term is 0 - 0: R8 without ever forming a difference of
// infinities.  `k0` = key index of the chunk's first column.
constexpr float kMaskedX = -1.0e30f;
template <bool RELU2, bool MASKED>
__device__ __forceinline__ void scale_chunk(const LogitChunk& c, float sc1, float sc2, float nm1, float nm2, XChunk& x, int k0, int limit) {
  const float2 vsc1 = make_float2(sc1, sc1), vsc2 = make_float2(sc2, sc2), vn1 = make_float2(nm1, nm1), vn2 = make_float2(nm2, nm2);
#pragma unroll
  for (int u = 0; u < 4; ++u) {
    x.x1[u] = fma2(make_float2(__uint_as_float(c.a[2 * u]), __uint_as_float(c.a[2 * u + 1])), vsc1, vn1);
    x.x2[u] = fma2(make_float2(__uint_as_float(c.b[2 * u]), __uint_as_float(c.b[2 * u + 1])), vsc2, vn2);
    if (RELU2) x.x2[u] = make_float2(fmaxf(x.x2[u].x, nm2), fmaxf(x.x2[u].y, nm2));
    if (MASKED) {
      const bool ok0 = k0 + 2 * u <= limit, ok1 = k0 + 2 * u + 1 <= limit;
      x.x1[u] = make_float2(ok0 ? x.x1[u].x : kMaskedX, ok1 ? x.x1[u].y : kMaskedX);
      x.x2[u] = make_float2(ok0 ? x.x2[u].x : kMaskedX, ok1 ? x.x2[u].y : kMaskedX);
    }
  }
}
// Compiler-level ordering point (no instruction): everything that uses x stays below the statements above this call --
// in particular below the tcgen05.ld that prefetches the next chunk.
__device__ __forceinline__ void pin_below(XChunk& x) {
  asm volatile("" : "+f"(x.x1[0].x), "+f"(x.x1[0].y), "+f"(x.x1[1].x), "+f"(x.x1[1].y), "+f"(x.x1[2].x), "+f"(x.x1[2].y), "+f"(x.x1[3].x),
                    "+f"(x.x1[3].y), "+f"(x.x2[0].x), "+f"(x.x2[0].y), "+f"(x.x2[1].x), "+f"(x.x2[1].y), "+f"(x.x2[2].x), "+f"(x.x2[2].y),
                    "+f"(x.x2[3].x), "+f"(x.x2[3].y));
}
// Alg.1 lines 10-12 for one unmasked chunk against the CURRENT reference (no row maximum, no alpha): bit u of PM sends
// column pair u's exps to the FMA-pipe polynomial.  FIRST: the step's first chunk starts the step-local sums.
template <uint32_t PM, bool FIRST>
__device__ __forceinline__ void accumulate_chunk(const XChunk& x, float2& T1, float2& T2, float2& TD) {
#pragma unroll
  for (int u = 0; u < 4; ++u) {
    const float2 x1 = x.x1[u], x2 = x.x2[u];
    const bool poly = (PM >> u) & 1u;
    const float2 p1 = poly ? ex2_poly2(x1) : make_float2(ex2_approx(x1.x), ex2_approx(x1.y));
    const float2 p2 = poly ? ex2_poly2(x2) : make_float2(ex2_approx(x2.x), ex2_approx(x2.y));
    if (FIRST && u == 0) {
      T1 = p1;
      T2 = p2;
      TD = mul2(p1, sub2(x1, x2));
    } else {
      T1 = add2(T1, p1);
      T2 = add2(T2, p2);
      TD = fma2(p1, sub2(x1, x2), TD);
    }
  }
}

// One whole step the careful way, Alg.1 lines 8-12 literally: row maximum over the visible keys of this thread's 32 columns,
// references raised to it, running sums rescaled by alpha (R9: alpha1 on R1, RD; alpha2 on R2), then every p <= 1.  Reads
// the logits from TMEM chunk by chunk, twice.  Used for masked steps (causal diagonal, key tails; MASKED) and to redo a
// step whose sums showed a stale reference.  `kbase` = key index of the thread's first column, `limit` = last visible key.
template <bool MASKED>
__device__ __noinline__ RowState safe_step(uint32_t taddr, RowState st, float sc1, float sc2, int kbase, int limit, bool relu2) {
  float mx1 = -CUDART_INF_F, mx2 = -CUDART_INF_F;
#pragma unroll 1
  for (int c = 0; c < 4; ++c) {
    LogitChunk ch;
    ld_chunk(taddr + c * 8, ch);
    wait_chunk(ch);
#pragma unroll
    for (int e = 0; e < 8; ++e) {
      const bool ok = !MASKED || (kbase + c * 8 + e) <= limit;
      mx1 = fmaxf(mx1, ok ? __uint_as_float(ch.a[e]) : -CUDART_INF_F);
      mx2 = fmaxf(mx2, ok ? (relu2 ? fmaxf(__uint_as_float(ch.b[e]), 0.f) : __uint_as_float(ch.b[e])) : -CUDART_INF_F);
    }
  }
  const float m1n = fmaxf(st.m1, mx1 * sc1), m2n = fmaxf(st.m2, mx2 * sc2);   // sc > 0: max commutes with the scale
  // R7: a row whose every key so far is masked keeps m = -inf; reference 0 so that (-inf) - (-inf) never forms
  const float ref1 = (m1n == -CUDART_INF_F) ? 0.f : m1n, ref2 = (m2n == -CUDART_INF_F) ? 0.f : m2n;
  const bool had1 = st.m1 != -CUDART_INF_F, had2 = st.m2 != -CUDART_INF_F;
  const float dm1 = had1 ? st.m1 - ref1 : 0.f, dm2 = had2 ? st.m2 - ref2 : 0.f;   // <= 0
  const float a1 = had1 ? ex2_approx(dm1) : 0.f, a2 = had2 ? ex2_approx(dm2) : 0.f;  // alpha (Alg.1 line 9)
  // x_t' = x_t + dm_t  =>  R1' = a1 R1,  R2' = a2 R2,  RD' = a1 (RD + (dm1 - dm2) R1)        (Eq.9-10 for the sums relative to m)
  const float dd = dm1 - dm2;
  st.RD = make_float2(a1 * fmaf(dd, st.R1.x, st.RD.x), a1 * fmaf(dd, st.R1.y, st.RD.y));
  st.R1 = make_float2(a1 * st.R1.x, a1 * st.R1.y);
  st.R2 = make_float2(a2 * st.R2.x, a2 * st.R2.y);
  st.m1 = m1n;
  st.m2 = m2n;
  float s1 = 0.f, s2 = 0.f, sd = 0.f;
#pragma unroll 1
  for (int c = 0; c < 4; ++c) {
    LogitChunk ch;
    ld_chunk(taddr + c * 8, ch);
    wait_chunk(ch);
#pragma unroll
    for (int e = 0; e < 8; ++e) {
      const float x1 = fmaf(__uint_as_float(ch.a[e]), sc1, -ref1);
      const float x2 = fmaf(relu2 ? fmaxf(__uint_as_float(ch.b[e]), 0.f) : __uint_as_float(ch.b[e]), sc2, -ref2);
      // R8: zero P~ at masked entries, take the difference from the raw (finite) logits
      const bool ok = !MASKED || (kbase + c * 8 + e) <= limit;
      const float p1 = ok ? ex2_approx(x1) : 0.f;
      const float p2 = ok ? ex2_approx(x2) : 0.f;
      s1 += p1;
      s2 += p2;
      sd = fmaf(p1, x1 - x2, sd);
    }
  }
  st.R1.x += s1;
  st.R2.x += s2;
  st.RD.x += sd;
  return st;   // by value: the state stays in registers across the call (a reference parameter would pin it to local memory)
}

// MC: launched as clusters of two CTAs that own the two Q tiles (2i, 2i+1) of one head and share ONE K stream -- each CTA's
// producer loads half of every stage's K-blocks and multicasts them into both CTAs' rings (half the L2 -> SM traffic per
// tile pair; SURVEY 8(f) NEXT-3 "2-CTA / multicast variants").  Both CTAs run the K pipeline for the pair's longer step
// count; a stage is reloaded only after BOTH issuers' MMAs on it have retired (k_empty counts two multicast commits).
// P2 (BLOCKED plan only): the two CTAs of a cluster pair issue ONE `tcgen05.mma.cta_group::2` per K-slice -- M = 256 (each CTA's
// 128 query rows, logits into each CTA's own TMEM), N = 128 keys of which each CTA holds 64 in its shared memory.  A K-block costs each
// CTA 8 KB instead of 16 (the ring beside a 128 KB Q tile is twice as deep, the L2 -> SM stream per CTA half as wide).  Rank 0 is
// the leader: its issuer warp issues every MMA, all TMA loads of both CTAs complete on ITS full barriers, its commits are multicast
// to both CTAs' k_empty / s_full, and both CTAs' softmax warps arrive on ITS s_empty.  Both CTAs run the pair's longer step count; a
// CTA past its own causal frontier sees fully masked steps.
template <int D1, int D2, bool CAUSAL, bool SPLIT = false, bool MC = false, bool P2 = false>
__global__ void __launch_bounds__(FwdCfg<D1, D2>::THREADS, 1)
streamkl_fwd_sm100_kernel(const __grid_constant__ CUtensorMap tmQ1, const __grid_constant__ CUtensorMap tmK1,
                          const __grid_constant__ CUtensorMap tmQ2, const __grid_constant__ CUtensorMap tmK2, const FwdParams p) {
  using C = FwdCfg<D1, D2>;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  const int KB1 = C::BLOCKED ? p.kb1 : C::KB1, KB2 = C::BLOCKED ? p.kb2 : C::KB2;
  const int NRING = C::BLOCKED ? p.nring : C::NSTAGE;      // ring entries: whole stages, or single K-blocks (BLOCKED)
  constexpr int SLOT_BYTES = P2 ? C::KBLK / 2 : C::STAGE_BYTES;   // P2: this CTA's 64 keys of a K-block
  constexpr bool PAIRED = MC || P2;
  uint8_t* sQ1 = smem;
  uint8_t* sQ2 = sQ1 + KB1 * C::QBLK;
  uint8_t* sK = smem + (KB1 + KB2) * C::QBLK;
  uint64_t* bars = reinterpret_cast<uint64_t*>(sK + NRING * SLOT_BYTES);
  uint64_t* q_full = bars;                    // 1
  uint64_t* k_full = bars + 1;                // NRING
  uint64_t* k_empty = k_full + NRING;         // NRING
  uint64_t* s_full = k_empty + NRING;         // 2 (TMEM stage written by the tensor pipe)
  uint64_t* s_empty = s_full + 2;             // 2 (all sixteen softmax warps are done with the stage)
  uint32_t* tmem_ptr = reinterpret_cast<uint32_t*>(s_empty + 2);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  // heavy (late, causal) query tiles first within each head; consecutive CTAs share a head (K stays in L2)
  static_assert(!(PAIRED && SPLIT) && !(MC && P2) && !(P2 && !C::BLOCKED), "the pair plans exist for the default grid; P2 for the BLOCKED plan");
  const int tile = SPLIT ? int(blockIdx.x) / p.W : (PAIRED ? int(blockIdx.x) >> 1 : int(blockIdx.x));
  const int wk = SPLIT ? int(blockIdx.x) % p.W : 0;          // key chunk of this CTA (split-K grid (b, i, w))
  const int crank = PAIRED ? int(blockIdx.x) & 1 : 0;        // rank within the cluster pair
  const int TQU = PAIRED ? (p.TQ + 1) / 2 : p.TQ;            // scheduling units per head: Q tiles, or pairs of them
  const int bh = tile / TQU;
  const int hq = bh % p.H, bq = bh / p.H, hk = hq / p.G;      // TMA coordinates {d, row, head, batch}
  // pairs: pair u (heavy first) = tiles TQ-1-2u (rank 0) and TQ-2-2u (rank 1; absent for the last pair of an odd TQ)
  const int qt_raw = PAIRED ? p.TQ - 1 - 2 * (tile % TQU) - crank : p.TQ - 1 - (tile % p.TQ);
  const bool has_tile = qt_raw >= 0;
  const int qt = (P2 && !has_tile) ? 0 : qt_raw;             // P2: an absent partner still consumes its TMEM stages: it recomputes tile 0, stores nothing
  const int q0 = qt * C::BQ;
  const int off = p.NK - p.NQ;
  const int TK = (p.NK + C::BK - 1) / C::BK;
  const int j_begin = SPLIT ? wk * p.chunk_steps : 0;        // this CTA's 128-key steps are [j_begin, j_begin + nsteps)
  int j_end = SPLIT ? min(TK, j_begin + p.chunk_steps) : TK;
  if (CAUSAL) j_end = min(j_end, min(p.NK - 1, q0 + C::BM - 1 + off) / C::BK + 1);   // past the tile's causal frontier
  // pairs: steps of the K pipeline both CTAs run = the pair's longer count (rank 0 owns the later tile: never the shorter one)
  int nsteps_pair = max(0, j_end - j_begin);
  if (PAIRED) {
    const int q0a = (qt_raw + crank) * C::BQ;                // rank 0's tile
    nsteps_pair = CAUSAL ? min(TK, min(p.NK - 1, q0a + C::BM - 1 + off) / C::BK + 1) : TK;
  }
  // MC: a CTA computes its own steps only (an absent partner none).  P2: the MMAs are the pair's, so every role of both CTAs runs the
  // pair's count (steps past a CTA's own frontier are fully masked for its rows)
  const int nsteps = P2 ? nsteps_pair : ((MC && !has_tile) ? 0 : max(0, j_end - j_begin));

  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tmQ1); tma_prefetch_desc(&tmK1); tma_prefetch_desc(&tmQ2); tma_prefetch_desc(&tmK2);
  }
  if (warp == 1 && lane == 0) {
    mbar_init(q_full, 1);
    for (int s = 0; s < NRING; ++s) { mbar_init(&k_full[s], 1); mbar_init(&k_empty[s], MC ? 2 : 1); }
    for (int i = 0; i < 2; ++i) { mbar_init(&s_full[i], 1); mbar_init(&s_empty[i], (P2 ? 2 : 1) * 4 * C::NGRP); }   // P2: both CTAs' softmax warps
    fence_mbar_init();
  }
  if (warp == 2) {
    if constexpr (P2) tmem_alloc_pair<C::TMEM_COLS>(tmem_ptr); else tmem_alloc<C::TMEM_COLS>(tmem_ptr);
  }
  tc_fence_before();
  __syncthreads();
  if (PAIRED) cluster_sync_all();   // the peer's barriers exist before anything is multicast to them
  tc_fence_after();
  const uint32_t tmem_base = *tmem_ptr;

  if (warp < 4) {
   reg_dealloc<24>();   // (pool: (96-24)*128 = 9216 >= (112-96)*512) producer / MMA / allocator warpgroup gives its registers to the softmax warpgroups
   if (warp == 0) {
    // ===================== TMA producer =====================
    if constexpr (P2) {
      if (lane == 0 && nsteps > 0) {
        const uint64_t pol_q = l2_policy_evict_first(), pol_k = l2_policy_evict_last();
        // every load of both CTAs completes on the LEADER's barrier, which expects both CTAs' bytes
        const uint32_t lq = mapa_shared(q_full, 0);
        if (crank == 0) mbar_arrive_expect_tx(q_full, uint32_t(2 * (KB1 + KB2) * C::QBLK));
        for (int kb = 0; kb < KB1; ++kb) tma_load_4d_pair(sQ1 + kb * C::QBLK, &tmQ1, lq, kb * 64, q0, hq, bq, pol_q);
        for (int kb = 0; kb < KB2; ++kb) tma_load_4d_pair(sQ2 + kb * C::QBLK, &tmQ2, lq, kb * 64, q0, hq, bq, pol_q);
        int slot = 0;
        uint32_t ph = 0;
        for (int j = 0; j < nsteps; ++j) {
          for (int b = 0; b < KB1 + KB2; ++b) {
            mbar_wait(&k_empty[slot], ph ^ 1);                       // (the leader's commit, multicast to both CTAs)
            if (crank == 0) mbar_arrive_expect_tx(&k_full[slot], uint32_t(2 * SLOT_BYTES));
            const bool one = b < KB1;
            // this CTA's 64 keys of the 128-key block (the K maps of this plan have 64-row boxes)
            tma_load_4d_pair(sK + slot * SLOT_BYTES, one ? &tmK1 : &tmK2, mapa_shared(&k_full[slot], 0), (one ? b : b - KB1) * 64,
                             j * C::BK + crank * (C::BK / 2), hk, bq, pol_k);
            if (++slot == NRING) { slot = 0; ph ^= 1; }
          }
        }
      }
    } else
    if (lane == 0 && (MC ? nsteps_pair : nsteps) > 0) {
      const uint64_t pol_q = l2_policy_evict_first(), pol_k = l2_policy_evict_last();
      if (nsteps > 0) {
        mbar_arrive_expect_tx(q_full, uint32_t((KB1 + KB2) * C::QBLK));
#pragma unroll
        for (int kb = 0; kb < KB1; ++kb) tma_load_4d_hint(sQ1 + kb * C::QBLK, &tmQ1, q_full, kb * 64, q0, hq, bq, pol_q);
#pragma unroll
        for (int kb = 0; kb < KB2; ++kb) tma_load_4d_hint(sQ2 + kb * C::QBLK, &tmQ2, q_full, kb * 64, q0, hq, bq, pol_q);
      }
      if constexpr (MC && C::BLOCKED) {
        // every CTA expects every block on its own barrier; it issues (and multicasts) the blocks of its own parity
        int slot = 0, cnt = 0;
        uint32_t ph = 0;
        for (int j = 0; j < nsteps_pair; ++j) {
          for (int b = 0; b < KB1 + KB2; ++b, ++cnt) {
            mbar_wait(&k_empty[slot], ph ^ 1);
            mbar_arrive_expect_tx(&k_full[slot], C::KBLK);
            const bool one = b < KB1;
            if ((cnt & 1) == crank)
              tma_load_4d_mcast(sK + slot * C::KBLK, one ? &tmK1 : &tmK2, &k_full[slot], (one ? b : b - KB1) * 64, j * C::BK, hk, bq, uint16_t(3),
                                pol_k);
            if (++slot == NRING) { slot = 0; ph ^= 1; }
          }
        }
        // drain: the last NRING blocks' release by both issuers (slot / ph now name the entry after the last one used)
        const int total = nsteps_pair * (KB1 + KB2);
        for (int i = 0; i < min(total, NRING); ++i) {
          mbar_wait(&k_empty[slot], ph ^ 1);
          if (++slot == NRING) { slot = 0; ph ^= 1; }
        }
      } else if constexpr (MC) {
        for (int j = 0; j < nsteps_pair; ++j) {
          const int s = j % C::NSTAGE;
          const uint32_t ph = (j / C::NSTAGE) & 1;
          mbar_wait(&k_empty[s], ph ^ 1);                       // both CTAs' MMAs on this stage have retired
          mbar_arrive_expect_tx(&k_full[s], C::STAGE_BYTES);    // the whole stage: this CTA's blocks and the peer's
          uint8_t* st = sK + s * C::STAGE_BYTES;
#pragma unroll
          for (int kb = 0; kb < C::KB1 + C::KB2; ++kb)
            if ((kb & 1) == crank)
              tma_load_4d_mcast(st + kb * C::KBLK, kb < C::KB1 ? &tmK1 : &tmK2, &k_full[s], (kb < C::KB1 ? kb : kb - C::KB1) * 64, j * C::BK, hk, bq,
                                uint16_t(3), pol_k);
        }
        // drain: the last commits of both issuers have arrived here before this CTA may leave the cluster
        for (int j = max(0, nsteps_pair - C::NSTAGE); j < nsteps_pair; ++j) mbar_wait(&k_empty[j % C::NSTAGE], (j / C::NSTAGE) & 1);
      } else
      if constexpr (C::BLOCKED) {
        // one ring entry per K-block, in the order the issuer consumes them: K1 blocks of step j, then its K2 blocks
        int slot = 0;
        uint32_t ph = 0;
        for (int j = 0; j < nsteps; ++j) {
          for (int b = 0; b < KB1 + KB2; ++b) {
            mbar_wait(&k_empty[slot], ph ^ 1);
            mbar_arrive_expect_tx(&k_full[slot], C::KBLK);
            const bool one = b < KB1;
            tma_load_4d_hint(sK + slot * C::KBLK, one ? &tmK1 : &tmK2, &k_full[slot], (one ? b : b - KB1) * 64, (j_begin + j) * C::BK, hk, bq,
                             pol_k);
            if (++slot == NRING) { slot = 0; ph ^= 1; }
          }
        }
      } else
      for (int j = 0; j < nsteps; ++j) {
        const int s = j % C::NSTAGE;
        const uint32_t ph = (j / C::NSTAGE) & 1;
        mbar_wait(&k_empty[s], ph ^ 1);
        mbar_arrive_expect_tx(&k_full[s], C::STAGE_BYTES);
        uint8_t* st = sK + s * C::STAGE_BYTES;
#pragma unroll
        for (int kb = 0; kb < C::KB1; ++kb)
          tma_load_4d_hint(st + kb * C::KBLK, &tmK1, &k_full[s], kb * 64, (j_begin + j) * C::BK, hk, bq, pol_k);
#pragma unroll
        for (int kb = 0; kb < C::KB2; ++kb)
          tma_load_4d_hint(st + (C::KB1 + kb) * C::KBLK, &tmK2, &k_full[s], kb * 64, (j_begin + j) * C::BK, hk, bq, pol_k);
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer =====================
    // The whole warp runs the loop (warp-uniform control flow and descriptors stay in uniform registers); only the
    // tcgen05.mma / tcgen05.commit instructions themselves are issued by one elected lane.
    const uint32_t idesc = umma_idesc_16(C::BM, C::BK, 0, 0, p.fmt16);
    const uint64_t dq1 = umma_smem_desc_sw128(smem_u32(sQ1), 16, 1024);
    const uint64_t dq2 = umma_smem_desc_sw128(smem_u32(sQ2), 16, 1024);
    const uint64_t dk = umma_smem_desc_sw128(smem_u32(sK), 16, 1024);
    if constexpr (P2) {
      if (crank == 0 && nsteps > 0) {       // the leader issues the pair's MMAs
        const uint32_t idesc2 = umma_idesc_16(2 * C::BM, C::BK, 0, 0, p.fmt16);
        mbar_wait(q_full, 0);
        tc_fence_after();
        int slot = 0;
        uint32_t ph = 0;
        for (int j = 0; j < nsteps; ++j) {
          const int st = j & 1;
          mbar_wait(&s_empty[st], ((j >> 1) & 1) ^ 1);       // both CTAs' softmax warps are done with the stage
          const uint32_t dS1 = tmem_base + st * (2 * C::BK);
          for (int b = 0; b < KB1 + KB2; ++b) {
            mbar_wait(&k_full[slot], ph);                    // both halves of the block have landed
            tc_fence_after();
            const bool one = b < KB1;
            const uint32_t first = (b == 0 || b == KB1) ? 0u : 1u;
            uint64_t a = dq1 + uint64_t((b * C::QBLK) >> 4), bk = dk + uint64_t((slot * SLOT_BYTES) >> 4);
            if (elect_one()) {
#pragma unroll
              for (int k = 0; k < 4; ++k)
                umma_bf16_ss_pair(one ? dS1 : dS1 + C::BK, a + uint64_t((k * 32) >> 4), bk + uint64_t((k * 32) >> 4), idesc2, first | uint32_t(k != 0));
              umma_commit_pair(&k_empty[slot], uint16_t(3));
              if (b + 1 == KB1 + KB2) umma_commit_pair(&s_full[st], uint16_t(3));
            }
            __syncwarp();
            if (++slot == NRING) { slot = 0; ph ^= 1; }
          }
        }
      }
    } else {
    if (nsteps > 0) {
      mbar_wait(q_full, 0);
      tc_fence_after();
    }
    if constexpr (C::BLOCKED) {
      int slot = 0;
      uint32_t ph = 0;
      for (int j = 0; j < (MC ? nsteps_pair : nsteps); ++j) {
        const int st = j & 1;
        const bool own = !MC || j < nsteps;   // MC: beyond this CTA's own steps only the shared ring is kept moving
        if (own) mbar_wait(&s_empty[st], ((j >> 1) & 1) ^ 1);
        const uint32_t dS1 = tmem_base + st * (2 * C::BK);
        for (int b = 0; b < KB1 + KB2; ++b) {
          mbar_wait(&k_full[slot], ph);
          tc_fence_after();
          if (!own) {
            if (elect_one()) umma_commit_mcast(&k_empty[slot], uint16_t(3));
            __syncwarp();
            if (++slot == NRING) { slot = 0; ph ^= 1; }
            continue;
          }
          const bool one = b < KB1;
          const uint32_t first = (b == 0 || b == KB1) ? 0u : 1u;        // a distribution's first block starts its accumulator
          uint64_t a = dq1 + uint64_t((b * C::QBLK) >> 4), bk = dk + uint64_t((slot * C::KBLK) >> 4);   // (Q2 blocks follow Q1's)
          if (elect_one()) {
#pragma unroll
            for (int k = 0; k < 4; ++k) umma_bf16_ss(one ? dS1 : dS1 + C::BK, a + uint64_t((k * 32) >> 4), bk + uint64_t((k * 32) >> 4), idesc, first | uint32_t(k != 0));
            // the block is reusable once these MMAs have retired (MC: in both CTAs)
            if (MC) umma_commit_mcast(&k_empty[slot], uint16_t(3)); else umma_commit(&k_empty[slot]);
            if (b + 1 == KB1 + KB2) umma_commit(&s_full[st]);
          }
          __syncwarp();
          if (++slot == NRING) { slot = 0; ph ^= 1; }
        }
      }
    } else
    for (int j = 0; j < (MC ? nsteps_pair : nsteps); ++j) {
      const int s = j % C::NSTAGE;
      const uint32_t ph = (j / C::NSTAGE) & 1;
      mbar_wait(&k_full[s], ph);
      if (MC && j >= nsteps) {   // the peer's tile is longer: keep the shared K pipeline moving, compute nothing
        if (elect_one()) umma_commit_mcast(&k_empty[s], uint16_t(3));
        __syncwarp();
        continue;
      }
      const int st = j & 1;
      const uint32_t sph = (j >> 1) & 1;
      mbar_wait(&s_empty[st], sph ^ 1);
      tc_fence_after();
      const uint32_t dS1 = tmem_base + st * (2 * C::BK);
      const uint32_t dS2 = dS1 + C::BK;
      // Per-step descriptor bases, laundered through an empty asm so that the sixteen A descriptors are formed as
      // base + immediate next to each MMA instead of being hoisted out of the loop (32 loop-invariant 64-bit values do
      // not fit this warp's register budget: ptxas spilled them and the issue loop, not the tensor pipe, set the pace).
      uint64_t a1 = dq1, a2 = dq2, bk = dk + uint64_t((s * C::STAGE_BYTES) >> 4);
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
        umma_commit(&s_full[st]);
        // K stage reusable once every MMA that read it has retired (MC: in both CTAs -- the arrive goes to both rings)
        if (MC) umma_commit_mcast(&k_empty[s], uint16_t(3)); else umma_commit(&k_empty[s]);
      }
      __syncwarp();
    }
    }   // (!P2)
   }
  } else {
    // ===================== softmax warps =====================
    reg_alloc<112>();    // needs 16*512 = 8192 registers from the pool the other warpgroup released
    const int quarter = warp & 3;          // TMEM lane quarter this warp may access
    const int grp = (warp - 4) >> 2;       // which 32-column group of every key tile (0 .. NGRP-1)
    const int rloc = quarter * 32 + lane;
    const int row = q0 + rloc;
    const int limit = CAUSAL ? min(p.NK - 1, row + off) : p.NK - 1;  // last visible key of this row
    // steps [0, n_fast) are unmasked for every row of this warp (key range of the group's 32 columns wholly visible to the
    // tile's first row and inside NK); the rest (causal diagonal, key tail) are masked.  Monotone in j.
    const int vis_all = CAUSAL ? min(p.NK - 1, q0 + off) : p.NK - 1;
    const int kg = vis_all - (C::BC - 1) - grp * C::BC;        // last admissible key index of a step's first column
    const int n_fast = kg < 0 ? 0 : max(0, min(nsteps, kg / C::BK + 1 - j_begin));
    const float sc1 = p.sc1, sc2 = p.sc2;
    const uint32_t tbase = tmem_base + (uint32_t(quarter * 32) << 16) + grp * C::BC;
    RowState st{-CUDART_INF_F, -CUDART_INF_F, make_float2(0.f, 0.f), make_float2(0.f, 0.f), make_float2(0.f, 0.f)};

    auto wait_full = [&](int j) {
      mbar_wait(&s_full[j & 1], (j >> 1) & 1);
      tc_fence_after();
    };
    auto release = [&](uint64_t* empty_bar) {   // every tcgen05.ld of this warp on the stage has completed (wait::ld)
      tc_fence_before();
      __syncwarp();
      if (lane == 0) {
        if (P2 && crank != 0) mbar_arrive_cluster(mapa_shared(empty_bar, 0));   // the pair's stage is free when BOTH CTAs are done: the leader counts
        else mbar_arrive(empty_bar);
      }
    };

    const bool relu2 = p.act2 == 1;
    // the fast loop, instantiated with and without the student's ReLU (chosen once per kernel: nothing on the hot path)
    auto run_fast = [&](auto relu_tag) {
      constexpr bool RELU2 = decltype(relu_tag)::value;
      LogitChunk A;
      XChunk X;
      wait_full(0);
      ld_chunk(tbase, A);
      wait_chunk(A);
      {
        // first tile of the row: take the reference from its first 8 columns (any finite reference will do; the check
        // below catches the case where the rest of the tile lies far above it)
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
      // One step on TMEM stage `tcur` (its first chunk already requested into A).  Per chunk: wait for the logits, turn
      // them into exponents (the only read of A), request the next chunk into A, then evaluate.  All addresses are stage
      // constants: the loop below is unrolled over the two stages.  `has_next`: another step follows (fast or masked) --
      // its first chunk is requested, after its s_full, before this step's last chunk is evaluated.
      // `masked_tag`: a step on the causal diagonal or the key tail (`k0` = key index of the thread's first column): the same
      // pipeline with the out-of-range keys neutralised in scale_chunk and every exp on MUFU (exact zeros).
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
        // the next step's logits have normally been in TMEM for a long time: probe its barrier now, use the answer after
        // this chunk's arithmetic (the probe's latency is then hidden)
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
        // warp-uniform decision: safe_step issues tcgen05.ld (.sync.aligned: the whole warp must execute it together);
        // a row that did not need the redo loses nothing by taking it
        if (!__any_sync(0xffffffffu, !(chk <= 1048576.f))) {   // (chk <= ... is false for inf / NaN)
          st.R1 = add2(st.R1, T1);            // Alg.1 lines 11-12 with alpha = 1
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
      uint32_t par = 0;   // parity of the s_full phases of the step pair (2i, 2i+1)
      int j = 0;
      for (; j + 2 <= n_fast; j += 2) {
        // (`has_next` is always true here, but it is kept a run-time value: the prefetch then sits in a basic block of its
        // own, ahead of the last chunk's arithmetic, instead of being sunk to the end of the step by the scheduler)
        fast_step(std::false_type{}, t0, t1, &s_full[1], par, &s_empty[0], j + 1 < nsteps, 0);
        fast_step(std::false_type{}, t1, t0, &s_full[0], par ^ 1, &s_empty[1], j + 2 < nsteps, 0);
        par ^= 1;
      }
      // what is left -- an odd unmasked step, then the masked steps (the row already has a reference) -- one step at a time
      for (; j < nsteps; ++j) {
        const uint32_t tc = (j & 1) ? t1 : t0, tn = (j & 1) ? t0 : t1;
        uint64_t* fn = &s_full[(j + 1) & 1];
        const uint32_t pn = uint32_t((j + 1) >> 1) & 1u;
        if (j < n_fast) fast_step(std::false_type{}, tc, tn, fn, pn, &s_empty[j & 1], j + 1 < nsteps, 0);
        else            fast_step(std::true_type{}, tc, tn, fn, pn, &s_empty[j & 1], j + 1 < nsteps, (j_begin + j) * C::BK + grp * C::BC);
      }
    };
    if (n_fast > 0) {   // (the group sees at least one whole unmasked step: every row has a finite reference before any masked step)
      if (relu2) run_fast(std::true_type{}); else run_fast(std::false_type{});
    } else {
      for (int j = 0; j < nsteps; ++j) {   // first Q tile of a causal head, NK < 128, ...: Alg.1 literally
        wait_full(j);
        st = safe_step<true>(tbase + (j & 1) * (2 * C::BK), st, sc1, sc2, (j_begin + j) * C::BK + grp * C::BC, limit, relu2);
        release(&s_empty[j & 1]);
      }
    }

    // this thread's partial statistics in Alg.1's form (log2 domain): l_t = R_t, acc = RD + (m1 - m2) R1
    const float pl1 = st.R1.x + st.R1.y, pl2 = st.R2.x + st.R2.y;
    const float pacc = (st.m1 == -CUDART_INF_F) ? 0.f : fmaf(st.m1 - st.m2, pl1, st.RD.x + st.RD.y);
    if (nsteps > 0) {
      // merge the column groups of each row (Eq.11 with (m2,l2) carried too, R11).  The exchange buffer aliases the Q1
      // block: every MMA that reads it has completed (the last s_full has been observed by every softmax warp).
      float* xch = reinterpret_cast<float*>(sQ1);
      if (grp > 0) {
        float* x = xch + (grp - 1) * 5 * C::BM;
        x[0 * C::BM + rloc] = st.m1; x[1 * C::BM + rloc] = pl1; x[2 * C::BM + rloc] = st.m2;
        x[3 * C::BM + rloc] = pl2; x[4 * C::BM + rloc] = pacc;
      }
      asm volatile("bar.sync 1, %0;" ::"n"(C::NGRP * 128) : "memory");
      if (grp == 0 && row < p.NQ && has_tile) {
        float m1 = st.m1, m2 = st.m2, l1 = pl1, l2 = pl2, acc = pacc;
#pragma unroll
        for (int hb = 1; hb < C::NGRP; ++hb) {
          const float* x = xch + (hb - 1) * 5 * C::BM;
          const float m1b = x[0 * C::BM + rloc], l1b = x[1 * C::BM + rloc], m2b = x[2 * C::BM + rloc];
          const float l2b = x[3 * C::BM + rloc], accb = x[4 * C::BM + rloc];
          const float n1 = fmaxf(m1, m1b), n2 = fmaxf(m2, m2b);
          // a group (or, split-K, a whole chunk) that lies past the row's causal frontier is (-inf, 0, 0): reference 0 (R7)
          const float r1 = (n1 == -CUDART_INF_F) ? 0.f : n1, r2 = (n2 == -CUDART_INF_F) ? 0.f : n2;
          const float wa1 = exp2f(m1 - r1), wb1 = exp2f(m1b - r1), wa2 = exp2f(m2 - r2), wb2 = exp2f(m2b - r2);
          l1 = l1 * wa1 + l1b * wb1; l2 = l2 * wa2 + l2b * wb2; acc = acc * wa1 + accb * wb1;
          m1 = n1; m2 = n2;
        }
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
    } else if (SPLIT && grp == 0 && row < p.NQ) {   // no step of this chunk is visible to this Q tile: identity partial
      float* o = p.part + (size_t(bh) * p.W + wk) * 5 * size_t(p.NQ) + row;
      o[0] = -CUDART_INF_F; o[size_t(p.NQ)] = 0.f; o[2 * size_t(p.NQ)] = -CUDART_INF_F; o[3 * size_t(p.NQ)] = 0.f;
      o[4 * size_t(p.NQ)] = 0.f;
    }
  }
  tc_fence_before();
  __syncthreads();
  if (PAIRED) cluster_sync_all();   // neither CTA leaves while the other may still write into its ring / TMEM or arrive on its barriers
  if (warp == 2) {
    tc_fence_after();
    if constexpr (P2) tmem_dealloc_pair<C::TMEM_COLS>(tmem_base); else tmem_dealloc<C::TMEM_COLS>(tmem_base);
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
