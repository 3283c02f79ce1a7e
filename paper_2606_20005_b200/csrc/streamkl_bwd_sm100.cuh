// streamkl_bwd_sm100.cuh -- StreamKL backward by recomputation for sm_100a.
//
// One kernel template, two instantiations per problem ("separate dQ / dK kernels", both
// deterministic and atomic-free because every output tile has exactly one owner):
//   OWNER_K = false : CTA owns a 128-row Q tile, streams 64-key tiles      -> dQ1, dQ2   (Alg.2 :224-234, Alg.3 :255-286)
//   OWNER_K = true  : CTA owns a 128-row K tile, streams 64-query tiles    -> dK1, dK2   (transposed tiling, :294, :309)
// With X the owner side and Y the streamed side, per step:
//   S1' = X1 Y1^T, S2' = X2 Y2^T        tcgen05.mma (SS) -> TMEM, lane = owner row                                (B2)
//   P_t = exp2(S_t' sc_t - lse_t log2e)  recomputed from the saved LSE (:216)                                     (B3)
//   dS2 = g (P2 - P1)   [fp32 subtract, one bf16 rounding]      dS1 = g P1 ((s1 - s2) - (lse1 - lse2) - kl)  Eq.12 (B4)
//   dX2 += dS2 Y2,  dX1 += dS1 Y1       tcgen05.mma with A = dS read FROM TMEM (the softmax warps write bf16 dS over
//                                        the logits they have just consumed, tcgen05.st), B = the Y tile in shared
//                                        memory read MN-major; accumulators stay in TMEM for the whole CTA         (B5)
// Epilogue: dX * c_t -> bf16 -> HBM, one rounding (B6).
//
// Everything is kept in the log2 domain: x_t = s_t' sc_t - lse_t log2e (sc_t = c_t log2e) so P_t = exp2(x_t) and
// (s1 - s2) - (lse1 - lse2) - kl = ln2 (x1 - x2 - kl log2e); the ln2 (and, for the Q owner, the per-row g) is folded
// into the epilogue scale.  Per-query scalars come from a small pre-pass (streamkl_bwd_stats_kernel) that writes, for
// every PAIR of queries, {-lse1 log2e (x2), -lse2 log2e (x2)}, {g (x2), kl log2e (x2)} -- the packed-fp32x2 operand
// layout -- padded to a multiple of 64 queries per head with values that make padded queries contribute exactly 0.
//
// Warp roles (640 threads): warp 0 TMA producer (X once, Y ring + the streamed queries' scalars when OWNER_K),
// warp 1 issues the S' MMAs, warp 3 issues the dX MMAs (two independent in-order streams into the tensor pipe, so a
// ready dX never queues behind an S' that waits for its TMEM stage and vice versa), warp 2 TMEM allocator,
// warps 4-19 sixteen dS warps = 2 step parities x 2 column halves x 4 TMEM lane quarters.
// TMEM (512 columns): NSS S' stages of {S1' 64, S2' 64}, released as soon as the dS warps hold the logits in registers;
// two dS stages of {dS1 32, dS2 32} packed-bf16 columns; D1 + D2 accumulator columns.  The two parity groups run
// decoupled: one group's TMEM load / store / barrier phases overlap the other group's exp phase.
#pragma once
#include <cuda_bf16.h>
#include <math_constants.h>

#include <type_traits>

#include "sm100_ptx.cuh"

// Share of the backward's exps evaluated by the FMA-pipe polynomial (ex2_poly2): one column pair in every N (0 = none),
// per kernel flavour.  Measured on B200: the student-only kernels are MUFU-bound (their tensor work is
// light) and gain 7-10 % from a quarter of the exps on the FMA pipe.  With teacher gradients the K owner alone gains
// (62.4 -> 57.3 ms on cfg 4) but draws more power, and under the 1000 W cap the forward and the Q owner then lose what it
// won (step 164.0 vs 163.8-165.6 ms): off.
#ifndef STREAMKL_BWD_POLY_STUDENT
#define STREAMKL_BWD_POLY_STUDENT 4
#endif
#ifndef STREAMKL_BWD_POLY_TEACHER_K
#define STREAMKL_BWD_POLY_TEACHER_K 0
#endif
#ifndef STREAMKL_BWD_POLY_TEACHER_Q
#define STREAMKL_BWD_POLY_TEACHER_Q 0
#endif

namespace skl {

template <int D1, int D2, bool TEACHER>
struct BwdCfg {
  static_assert(D1 % 64 == 0 && D2 % 64 == 0 && D1 <= 128 && D2 <= 128, "tcgen05 path: d in {64,128}");
  static constexpr int BX = 128;   // owner rows per CTA (TMEM lanes)
  static constexpr int BY = 64;    // streamed rows per step
  static constexpr int KB1 = D1 / 64, KB2 = D2 / 64;
  static constexpr int XBLK = BX * 128, YBLK = BY * 128;
  static constexpr int X_BYTES = (KB1 + KB2) * XBLK;
  static constexpr int Y_STAGE = (KB1 + KB2) * YBLK;
  static constexpr int STAT_STAGE = BY * 16;                         // two float4 per PAIR of streamed queries (OWNER_K)
  static constexpr int AUX_BYTES = 512;
  static constexpr int NSTAGE_RAW = (227 * 1024 - 1024 - AUX_BYTES - X_BYTES) / (Y_STAGE + STAT_STAGE);
  static constexpr int NSTAGE = NSTAGE_RAW > 6 ? 6 : NSTAGE_RAW;
  static_assert(NSTAGE >= 2, "need at least a double-buffered Y ring");
  static constexpr int SMEM_BYTES = 1024 + X_BYTES + NSTAGE * (Y_STAGE + STAT_STAGE) + AUX_BYTES;
  static constexpr int THREADS = 128 + 512;
  static constexpr uint32_t TMEM_COLS = 512;
  static constexpr int DX_COLS = D2 + (TEACHER ? D1 : 0);
  static constexpr int NSS = (512 - 128 - DX_COLS) / 128 >= 2 ? 2 : 1;           // S' stages that fit beside dS and dX
  static constexpr uint32_t COL_DS = NSS * 128;                                   // 2 stages x {dS1 32, dS2 32}
  static constexpr uint32_t COL_DX1 = COL_DS + 128, COL_DX2 = COL_DX1 + (TEACHER ? D1 : 0);
  static_assert(COL_DX2 + D2 <= 512, "TMEM budget");
};

// queries per head in the padded per-query scalar array
__host__ __device__ constexpr long long bwd_stats_padded_rows(long long NQ) { return (NQ + 63) / 64 * 64; }

// Element strides {batch, head, row} of a gradient tensor (the head dimension is contiguous) and its true head dim: the kernels
// run on head dims padded to 64 / 128 (TMA zero-fills the extra columns of the inputs); columns >= d are not stored.
struct OutGeom {
  long long sb, sh, sn;
  int d;
};
struct BwdParams {
  int NQ, NK, TX, BH;   // BH = B * H query heads
  int H, HK, G;         // query heads, K heads (H = HK * G), query heads per K head (GQA)
  uint32_t fmt16;       // 16-bit element format of inputs and gradients: 1 bf16, 0 fp16
  int act2;             // student activation: 0 none, 1 relu (s2 = relu(c2 <q2,k2>), R23): gates dS2 with relu'
  float c1, c2;
  const float4* stats;  // [B*H][NQP/2][2] float4, NQP = bwd_stats_padded_rows(NQ)
  uint16_t* dX1;        // dQ1 or dK1 (nullptr when !TEACHER), 16-bit elements
  uint16_t* dX2;        // dQ2 or dK2
  OutGeom g1, g2;
};

// B1: per-query scalars in the layout the dS warps consume (see the header comment)
static __global__ void streamkl_bwd_stats_kernel(const float* __restrict__ kl, const float* __restrict__ lse1, const float* __restrict__ lse2,
                                          const float* __restrict__ dkl, float4* __restrict__ stats, int NQ, long long pairs_per_head,
                                          long long total_pairs) {
  const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= total_pairs) return;
  const long long bh = idx / pairs_per_head;
  const int q = int(idx % pairs_per_head);
  const float L2E = 1.4426950408889634f;
  float v[2][4];
#pragma unroll
  for (int u = 0; u < 2; ++u) {
    const int i = 2 * q + u;
    if (i < NQ) {
      const size_t o = size_t(bh) * NQ + i;
      v[u][0] = -lse1[o] * L2E; v[u][1] = -lse2[o] * L2E; v[u][2] = dkl[o]; v[u][3] = kl[o] * L2E;
    } else {  // padded query: P = exp2(x - 1e30) = 0 and g = 0
      v[u][0] = -1e30f; v[u][1] = -1e30f; v[u][2] = 0.f; v[u][3] = 0.f;
    }
  }
  stats[idx * 2 + 0] = make_float4(v[0][0], v[1][0], v[0][1], v[1][1]);
  stats[idx * 2 + 1] = make_float4(v[0][2], v[1][2], v[0][3], v[1][3]);
}

__device__ __forceinline__ uint32_t pack_bf16x2(float lo, float hi) {
  uint32_t r;
  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
  return r;
}
__device__ __forceinline__ uint32_t pack_f16x2(float lo, float hi) {
  uint32_t r;
  asm("cvt.rn.f16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
  return r;
}
template <bool F16> __device__ __forceinline__ uint32_t pack_16x2(float lo, float hi) { return F16 ? pack_f16x2(lo, hi) : pack_bf16x2(lo, hi); }

// dX accumulator (this warp's 32 lanes x NC fp32 columns starting at column `col0`) -> * scale -> 16-bit -> global row;
// 8-column chunks at or beyond the true head dim `d` (a multiple of 8) are padding and are not stored
template <int NC>
__device__ __forceinline__ void store_dx_cols(uint32_t taddr, float scale, uint16_t* out, bool valid, bool f16, int col0, int d) {
  static_assert(NC == 16 || NC == 32, "column slice per dS warp group");
  uint32_t v[NC];
  if constexpr (NC == 32) tmem_ld32(taddr, v); else tmem_ld16(taddr, v);
  tmem_wait_ld();
  if (valid) {
#pragma unroll
    for (int q = 0; q < NC / 8; ++q) {
      if (col0 + q * 8 >= d) break;
      uint4 o;
      if (f16) {
        o.x = pack_f16x2(__uint_as_float(v[q * 8 + 0]) * scale, __uint_as_float(v[q * 8 + 1]) * scale);
        o.y = pack_f16x2(__uint_as_float(v[q * 8 + 2]) * scale, __uint_as_float(v[q * 8 + 3]) * scale);
        o.z = pack_f16x2(__uint_as_float(v[q * 8 + 4]) * scale, __uint_as_float(v[q * 8 + 5]) * scale);
        o.w = pack_f16x2(__uint_as_float(v[q * 8 + 6]) * scale, __uint_as_float(v[q * 8 + 7]) * scale);
      } else {
        o.x = pack_bf16x2(__uint_as_float(v[q * 8 + 0]) * scale, __uint_as_float(v[q * 8 + 1]) * scale);
        o.y = pack_bf16x2(__uint_as_float(v[q * 8 + 2]) * scale, __uint_as_float(v[q * 8 + 3]) * scale);
        o.z = pack_bf16x2(__uint_as_float(v[q * 8 + 4]) * scale, __uint_as_float(v[q * 8 + 5]) * scale);
        o.w = pack_bf16x2(__uint_as_float(v[q * 8 + 6]) * scale, __uint_as_float(v[q * 8 + 7]) * scale);
      }
      *reinterpret_cast<uint4*>(out + q * 8) = o;
    }
  }
}

__device__ __forceinline__ float4 lds_f4(uint32_t saddr) {
  float4 v;
  asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(saddr));
  return v;
}

// B3 + B4 for one owner row and NC streamed columns: logits r1,r2 (fp32 bits) -> packed bf16 dS1 (o1), dS2 (o2).
//   OWNER_Q: the row's scalars (nL1,nL2,klog) are thread constants and g is applied in the epilogue.
//   OWNER_K: per-column scalars come from shared memory (`stat`: shared-space address of these NC/2 column
//            pairs, two float4 each), g is applied here.
// MASKED: causal diagonal tiles and streamed-key tails; P (possibly inf for a zero-filled logit) is discarded by SELECT.
// RELU2 (R23): the student's logit is relu(s2'), i.e. x2 = max(x2_raw, -lse2 log2e) in the shifted log2 domain,
// and relu' = 1[<q2,k2> > 0] gates dS2.
template <int NC, bool TEACHER, bool OWNER_K, bool CAUSAL, bool MASKED, bool WANT2 = true, bool F16 = false, bool RELU2 = false>
__device__ __forceinline__ void ds_row(const uint32_t (&r1)[NC], const uint32_t (&r2)[NC], uint32_t (&o1)[NC / 2], uint32_t (&o2)[NC / 2],
                                         float sc1, float sc2, float nL1, float nL2, float klog, uint32_t stat, int xrow,
                                         int y0, int off, int NK) {
  const float2 vsc1 = make_float2(sc1, sc1), vsc2 = make_float2(sc2, sc2);
  float2 vn1 = make_float2(nL1, nL1), vn2 = make_float2(nL2, nL2), vk = make_float2(klog, klog), vg = make_float2(1.f, 1.f);
#pragma unroll
  for (int e = 0; e < NC; e += 2) {
    if constexpr (OWNER_K) {
      const float4 a = lds_f4(stat + e * 16), b = lds_f4(stat + e * 16 + 16);   // pair e/2: two float4
      vn1 = make_float2(a.x, a.y); vn2 = make_float2(a.z, a.w); vg = make_float2(b.x, b.y); vk = make_float2(b.z, b.w);
    }
    const float2 x1 = fma2(make_float2(__uint_as_float(r1[e]), __uint_as_float(r1[e + 1])), vsc1, vn1);
    float2 x2 = fma2(make_float2(__uint_as_float(r2[e]), __uint_as_float(r2[e + 1])), vsc2, vn2);
    bool on0 = true, on1 = true;
    if constexpr (RELU2) {
      // relu' on the sign of the raw accumulator (exact: sc2 > 0).  Comparing the shifted values instead would switch off a small
      // positive logit whose product with sc2 rounds away against |lse2 log2e|, where the definition 1[s2 > 0] keeps it on.
      on0 = __uint_as_float(r2[e]) > 0.f; on1 = __uint_as_float(r2[e + 1]) > 0.f;
      x2 = make_float2(fmaxf(x2.x, vn2.x), fmaxf(x2.y, vn2.y));
    }
    // P_t = exp(s_t - lse_t) (Alg.2 line 7); one column pair in every STREAMKL_BWD_POLY_EVERY on the FMA/ALU pipes
    constexpr int PE = TEACHER ? (OWNER_K ? STREAMKL_BWD_POLY_TEACHER_K : STREAMKL_BWD_POLY_TEACHER_Q) : STREAMKL_BWD_POLY_STUDENT;
    const bool poly = PE > 0 && ((e >> 1) % (PE > 0 ? PE : 1)) == 0;
    const float2 p1 = poly ? ex2_poly2(x1) : make_float2(ex2_approx(x1.x), ex2_approx(x1.y));
    const float2 p2 = poly ? ex2_poly2(x2) : make_float2(ex2_approx(x2.x), ex2_approx(x2.y));
    float2 a2 = make_float2(0.f, 0.f);
    if constexpr (WANT2) {
      a2 = sub2(p2, p1);                                                 // dS2 / g (Alg.2 line 8): fp32 subtract, rounded once below
      if constexpr (OWNER_K) a2 = mul2(a2, vg);
      if constexpr (RELU2) { a2.x = on0 ? a2.x : 0.f; a2.y = on1 ? a2.y : 0.f; }
    }
    float2 a1 = make_float2(0.f, 0.f);
    if constexpr (TEACHER) {                                             // dS1 / (g ln2) = P1 (x1 - x2 - kl log2e)   (Alg.3 lines 9-10, Eq.12)
      const float2 d = sub2(sub2(x1, x2), vk);
      a1 = mul2(OWNER_K ? mul2(p1, vg) : p1, d);
    }
    if constexpr (MASKED) {
      const int y = y0 + e;
      bool ok0, ok1;
      if constexpr (OWNER_K) { ok0 = (xrow < NK) && (!CAUSAL || xrow <= y + off); ok1 = (xrow < NK) && (!CAUSAL || xrow <= y + 1 + off); }
      else { ok0 = (y < NK) && (!CAUSAL || y <= xrow + off); ok1 = (y + 1 < NK) && (!CAUSAL || y + 1 <= xrow + off); }
      a2.x = ok0 ? a2.x : 0.f; a2.y = ok1 ? a2.y : 0.f;
      a1.x = ok0 ? a1.x : 0.f; a1.y = ok1 ? a1.y : 0.f;
    }
    if constexpr (WANT2) o2[e >> 1] = pack_16x2<F16>(a2.x, a2.y);
    if constexpr (TEACHER) o1[e >> 1] = pack_16x2<F16>(a1.x, a1.y);
  }
}


// three warp-uniform run-time flags -> compile-time tags (one branch tree per step; nothing inside ds_row's loop)
template <class F>
__device__ __forceinline__ void dispatch3(bool a, bool b, bool c, F&& f) {
  using T = std::true_type;
  using N = std::false_type;
  if (a) { if (b) { if (c) f(T{}, T{}, T{}); else f(T{}, T{}, N{}); } else { if (c) f(T{}, N{}, T{}); else f(T{}, N{}, N{}); } }
  else   { if (b) { if (c) f(N{}, T{}, T{}); else f(N{}, T{}, N{}); } else { if (c) f(N{}, N{}, T{}); else f(N{}, N{}, N{}); } }
}

template <int D1, int D2, bool CAUSAL, bool TEACHER, bool OWNER_K>
__global__ void __launch_bounds__(BwdCfg<D1, D2, TEACHER>::THREADS, 1)
streamkl_bwd_sm100_kernel(const __grid_constant__ CUtensorMap tmQ1, const __grid_constant__ CUtensorMap tmK1,
                          const __grid_constant__ CUtensorMap tmQ2, const __grid_constant__ CUtensorMap tmK2, const BwdParams p) {
  using C = BwdCfg<D1, D2, TEACHER>;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t* sX1 = smem;
  uint8_t* sX2 = sX1 + C::KB1 * C::XBLK;
  uint8_t* sY = smem + C::X_BYTES;                        // NSTAGE x {Y1 blocks, Y2 blocks}
  float4* sStat = reinterpret_cast<float4*>(sY + C::NSTAGE * C::Y_STAGE);   // NSTAGE x 64 float4
  uint64_t* bars = reinterpret_cast<uint64_t*>(reinterpret_cast<uint8_t*>(sStat) + C::NSTAGE * C::STAT_STAGE);
  uint64_t* x_full = bars;                       // 1
  uint64_t* y_full = bars + 1;                   // NSTAGE  (TMA bytes landed)
  uint64_t* y_empty = y_full + C::NSTAGE;        // NSTAGE  (count 2: the S' MMAs and the dX MMAs that read the stage have retired)
  uint64_t* s_full = y_empty + C::NSTAGE;        // 2  (per parity group) logits of the group's next step are in TMEM
  uint64_t* s_empty = s_full + 2;                // 2  (per parity group) its 8 dS warps hold those logits in registers
  uint64_t* ds_full = s_empty + 2;               // 2  dS stage written by its 8 dS warps
  uint64_t* ds_empty = ds_full + 2;              // 2  dS stage consumed by the dX MMAs
  uint64_t* dx_full = ds_empty + 2;              // 1
  uint32_t* tmem_ptr = reinterpret_cast<uint32_t*>(dx_full + 1);

  const CUtensorMap* tmX1 = OWNER_K ? &tmK1 : &tmQ1;
  const CUtensorMap* tmX2 = OWNER_K ? &tmK2 : &tmQ2;
  const CUtensorMap* tmY1 = OWNER_K ? &tmQ1 : &tmK1;
  const CUtensorMap* tmY2 = OWNER_K ? &tmQ2 : &tmK2;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  // the CTA's unit = (batch, owner head): a query head for the Q owner; a K head for the K owner, which then streams the
  // query tiles of all G query heads that share it (GQA; G = 1 otherwise).  TMA coordinates are {d, row, head, batch}.
  const int unit = blockIdx.x / p.TX;
  const int HX = OWNER_K ? p.HK : p.H;
  const int bx = unit / HX, hx = unit % HX;
  // heavy tiles first: late Q tiles see more keys, early K tiles are seen by more queries
  const int xt = (CAUSAL && !OWNER_K) ? (p.TX - 1 - (blockIdx.x % p.TX)) : (blockIdx.x % p.TX);
  const int x0 = xt * C::BX;
  const int off = p.NK - p.NQ;
  const int NX = OWNER_K ? p.NK : p.NQ;
  const int NY = OWNER_K ? p.NQ : p.NK;
  const long long NQP = bwd_stats_padded_rows(p.NQ);
  int j_begin = 0, j_end = (NY + C::BY - 1) / C::BY;
  if (CAUSAL) {
    if (OWNER_K) j_begin = max(0, x0 - off) / C::BY;                       // first query that sees key x0
    else         j_end = min(p.NK - 1, x0 + C::BX - 1 + off) / C::BY + 1;   // last key the tile's last row sees
  }
  const int nsteps1 = max(0, j_end - j_begin);             // steps per streamed head
  const int nsteps = nsteps1 * (OWNER_K ? p.G : 1);
  // step `it` -> (streamed head index g within the group, streamed tile j)
  auto step_g = [&](int it) { return OWNER_K ? it / max(nsteps1, 1) : 0; };
  auto step_j = [&](int it) { return j_begin + (OWNER_K ? it % max(nsteps1, 1) : it); };

  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tmQ1); tma_prefetch_desc(&tmK1); tma_prefetch_desc(&tmQ2); tma_prefetch_desc(&tmK2);
  }
  if (warp == 1 && lane == 0) {
    mbar_init(x_full, 1);
    for (int s = 0; s < C::NSTAGE; ++s) { mbar_init(&y_full[s], 1); mbar_init(&y_empty[s], 2); }
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
    reg_dealloc<32>();   // producer / MMA / allocator warpgroup gives its registers to the sixteen dS warps: 128*(96-32) = 512*(112-96)
    if (warp == 0) {
      // ===================== producer =====================
      if (lane == 0) {
        const uint64_t pol_x = l2_policy_evict_first(), pol_y = l2_policy_evict_last();
        mbar_arrive_expect_tx(x_full, C::X_BYTES);
#pragma unroll
        for (int kb = 0; kb < C::KB1; ++kb) tma_load_4d_hint(sX1 + kb * C::XBLK, tmX1, x_full, kb * 64, x0, hx, bx, pol_x);
#pragma unroll
        for (int kb = 0; kb < C::KB2; ++kb) tma_load_4d_hint(sX2 + kb * C::XBLK, tmX2, x_full, kb * 64, x0, hx, bx, pol_x);
        for (int it = 0; it < nsteps; ++it) {
          const int j = step_j(it);
          const int hy = OWNER_K ? hx * p.G + step_g(it) : hx / p.G;   // streamed head: a query head of the group / the K head
          const int s = it % C::NSTAGE;
          const uint32_t ph = (it / C::NSTAGE) & 1;
          mbar_wait(&y_empty[s], ph ^ 1);
          mbar_arrive_expect_tx(&y_full[s], C::Y_STAGE + (OWNER_K ? C::STAT_STAGE : 0));
          uint8_t* st = sY + s * C::Y_STAGE;
#pragma unroll
          for (int kb = 0; kb < C::KB1; ++kb) tma_load_4d_hint(st + kb * C::YBLK, tmY1, &y_full[s], kb * 64, j * C::BY, hy, bx, pol_y);
#pragma unroll
          for (int kb = 0; kb < C::KB2; ++kb)
            tma_load_4d_hint(st + (C::KB1 + kb) * C::YBLK, tmY2, &y_full[s], kb * 64, j * C::BY, hy, bx, pol_y);
          if (OWNER_K)   // the streamed queries' scalars (B1): 64 queries = 32 pairs x 32 B, contiguous and 1 KB aligned
            bulk_load_1d(sStat + s * C::BY, p.stats + (size_t(bx * p.H + hy) * NQP + size_t(j) * C::BY), C::STAT_STAGE, &y_full[s]);
        }
      }
    } else if (warp == 1) {
      // ===================== S' MMA issuer =====================
      // The whole warp runs the loop (warp-uniform control flow); only the tcgen05 instructions are issued by one lane.
      const uint32_t idesc_s = umma_idesc_16(C::BX, C::BY, 0, 0, p.fmt16);     // S' = X Y^T   : A,B K-major from smem
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
        const int prev = it - C::NSS;                    // the step whose logits this S' stage held last
        mbar_wait(&y_full[s], (it / C::NSTAGE) & 1);
        // s_full / s_empty are indexed by the PARITY GROUP that consumes the step (not by the stage), so that each
        // barrier is observed phase by phase by one group: a parity wait cannot tell phase n from phase n+2
        if (prev >= 0) mbar_wait(&s_empty[prev & 1], (prev >> 1) & 1);   // those logits are in registers
        tc_fence_after();
        uint64_t dys = dyk + uint64_t((s * C::Y_STAGE) >> 4), a1 = dx1, a2 = dx2;
        // launder the descriptor bases: every MMA's descriptors are then formed as base + immediate beside it instead
        // of sixteen loop-invariant 64-bit values being hoisted (and spilled: this warp runs on 32 registers)
        asm volatile("" : "+l"(a1), "+l"(a2), "+l"(dys));
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
          umma_commit(&y_empty[s]);     // first of the two arrivals that free the Y stage
        }
        __syncwarp();
      }
    } else if (warp == 3) {
      // ===================== dX MMA issuer =====================
      const uint32_t idesc_g1 = umma_idesc_16(C::BX, D1, 0, 1, p.fmt16);       // dX1 += dS1 Y1: A from TMEM, B MN-major
      const uint32_t idesc_g2 = umma_idesc_16(C::BX, D2, 0, 1, p.fmt16);
      // Y as the MN-major B operand: 64-column chunks YBLK apart (LBO), 8-row groups 1024 B apart (SBO);
      // a K=16 slice = 16 streamed rows = 2048 B
      const uint64_t dym = umma_smem_desc_sw128(smem_u32(sY), C::YBLK, 1024);
      for (int it = 0; it < nsteps; ++it) {
        const int s = it % C::NSTAGE;
        const int st = it & 1;
        mbar_wait(&ds_full[st], (it >> 1) & 1);   // implies the Y stage is resident (its S' MMAs ran before the dS warps did)
        tc_fence_after();
        uint64_t dys = dym + uint64_t((s * C::Y_STAGE) >> 4);
        asm volatile("" : "+l"(dys));
        const uint32_t tA = tmem_base + C::COL_DS + st * 64;
        const uint32_t acc = it > 0;
        if (elect_one()) {
          // K-slice k (16 streamed rows) of dS = 8 packed-bf16 TMEM columns
#pragma unroll
          for (int k = 0; k < 4; ++k)
            umma_bf16_ts(tmem_base + C::COL_DX2, tA + 32 + k * 8, dys + uint64_t((C::KB1 * C::YBLK + k * 2048) >> 4), idesc_g2,
                         acc | (k != 0));
          if (TEACHER) {
#pragma unroll
            for (int k = 0; k < 4; ++k)
              umma_bf16_ts(tmem_base + C::COL_DX1, tA + k * 8, dys + uint64_t((k * 2048) >> 4), idesc_g1, acc | (k != 0));
          }
          umma_commit(&ds_empty[st]);
          umma_commit(&y_empty[s]);     // second arrival
          if (it + 1 == nsteps) umma_commit(dx_full);
        }
        __syncwarp();
      }
    }
  } else {
    // ===================== dS warps =====================
    reg_alloc<112>();
    const int sw = warp - 4;
    const int quarter = warp & 3;             // TMEM lane quarter this warp may access
    const int grp = sw >> 2;                  // 0..3
    const int par = grp & 1;                  // this warp group takes the steps of that parity (= its dS stage)
    const int half = grp >> 1;                // 32-column half of every streamed tile
    const int rloc = quarter * 32 + lane;     // owner row within the tile = TMEM lane
    const int xrow = x0 + rloc;
    const float L2E = 1.4426950408889634f, LN2 = 0.6931471805599453f;
    const float sc1 = p.c1 * L2E, sc2 = p.c2 * L2E;
    float nL1 = -1e30f, nL2 = -1e30f, klog = 0.f, my_g = 0.f;
    if (!OWNER_K && xrow < p.NQ) {
      const float* sp = reinterpret_cast<const float*>(p.stats + (size_t(unit) * NQP + size_t(xrow & ~1)));  // pair (xrow>>1): 2 float4
      const int u = xrow & 1;
      nL1 = sp[u]; nL2 = sp[2 + u]; my_g = sp[4 + u]; klog = sp[6 + u];
    }
    const uint32_t lane_addr = tmem_base + (uint32_t(quarter * 32) << 16);
    const uint32_t stat_base = smem_u32(sStat) + half * 32 * 16;
    const uint32_t ds_addr = lane_addr + C::COL_DS + par * 64 + half * 16;   // dS1 here, dS2 32 columns further
    const bool f16 = p.fmt16 == 0, relu2 = p.act2 == 1;
    for (int it = par; it < nsteps; it += 2) {
      const int j = step_j(it);
      const int s = it % C::NSTAGE;
      const int ss = it % C::NSS;
      mbar_wait(&s_full[par], (it >> 1) & 1);
      tc_fence_after();
      const uint32_t taddr = lane_addr + ss * 128 + half * 32;
      uint32_t r1[32], r2[32], o1[16], o2[16];
      tmem_ld32(taddr, r1);
      tmem_ld32(taddr + 64, r2);
      tmem_wait_ld();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&s_empty[par]);   // logits are in registers: the next S' may overwrite this stage
      const int y0 = j * C::BY + half * 32;
      // warp-uniform: does any (query,key) pair of this 128 x 32 block fall outside the mask?
      // (a streamed KEY tail is masked too: TMA zero-fills those rows, but P = exp2(0 - lse) may overflow)
      const bool masked = OWNER_K ? (CAUSAL && (y0 + off < x0 + C::BX - 1))
                                  : ((CAUSAL && (y0 + 31 > x0 + off)) || (y0 + 32 > p.NK));
      const uint32_t stat = stat_base + s * C::STAT_STAGE;
      dispatch3(masked, f16, relu2, [&](auto m, auto h, auto r) {
        ds_row<32, TEACHER, OWNER_K, CAUSAL, decltype(m)::value, true, decltype(h)::value, decltype(r)::value>(
            r1, r2, o1, o2, sc1, sc2, nL1, nL2, klog, stat, xrow, y0, off, p.NK);
      });
      mbar_wait(&ds_empty[par], ((it >> 1) & 1) ^ 1);   // the dX MMAs of step it-2 have consumed this dS stage
      tc_fence_after();
      tmem_st16(ds_addr + 32, o2);
      if (TEACHER) tmem_st16(ds_addr, o1);
      tmem_wait_st();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&ds_full[par]);
    }
    // ---- epilogue: dX (TMEM fp32) * c_t -> 16-bit -> HBM; each warp group takes a quarter of the (padded) columns
    const bool valid = xrow < NX;
    const long long xr = valid ? xrow : 0;
    uint16_t* o2 = p.dX2 + (bx * p.g2.sb + hx * p.g2.sh + xr * p.g2.sn) + grp * (D2 / 4);
    uint16_t* o1 = TEACHER ? p.dX1 + (bx * p.g1.sb + hx * p.g1.sh + xr * p.g1.sn) + grp * (D1 / 4) : nullptr;
    const float g_row = OWNER_K ? 1.f : my_g;   // Q owner: g is a per-row factor of dS, applied here
    if (nsteps > 0) {
      mbar_wait(dx_full, 0);
      tc_fence_after();
      store_dx_cols<D2 / 4>(lane_addr + C::COL_DX2 + grp * (D2 / 4), p.c2 * g_row, o2, valid, f16, grp * (D2 / 4), p.g2.d);
      if (TEACHER) store_dx_cols<D1 / 4>(lane_addr + C::COL_DX1 + grp * (D1 / 4), p.c1 * LN2 * g_row, o1, valid, f16, grp * (D1 / 4), p.g1.d);
    } else if (valid) {
      const uint4 z = make_uint4(0, 0, 0, 0);
      for (int c = 0; c < D2 / 4 && grp * (D2 / 4) + c < p.g2.d; c += 8) *reinterpret_cast<uint4*>(o2 + c) = z;
      if (TEACHER) for (int c = 0; c < D1 / 4 && grp * (D1 / 4) + c < p.g1.d; c += 8) *reinterpret_cast<uint4*>(o1 + c) = z;
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
