// streamkl_simt.cuh -- fp32 CUDA-core kernels for the cases the tcgen05 path does not cover:
// fp32 inputs (config 1 of BASELINE.json needs >= tf32 operand precision, R17) and head dims other
// than {64,128}.  Same algorithms (Alg.1 forward with a 1-key "tile", Alg.2/3 and their K-owner transposes),
// organised as "one thread owns one row": the owner's rows live in padded shared memory, the other side is
// streamed through shared memory in 32-row tiles, every update is thread-local (no reductions, no atomics).
#pragma once
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <math_constants.h>

namespace skl {

template <typename T> __device__ __forceinline__ float to_f32(T v);
template <> __device__ __forceinline__ float to_f32<float>(float v) { return v; }
template <> __device__ __forceinline__ float to_f32<__nv_bfloat16>(__nv_bfloat16 v) { return __bfloat162float(v); }
template <> __device__ __forceinline__ float to_f32<__half>(__half v) { return __half2float(v); }
template <typename T> __device__ __forceinline__ T from_f32(float v);
template <> __device__ __forceinline__ float from_f32<float>(float v) { return v; }
template <> __device__ __forceinline__ __nv_bfloat16 from_f32<__nv_bfloat16>(float v) { return __float2bfloat16_rn(v); }
template <> __device__ __forceinline__ __half from_f32<__half>(float v) { return __float2half_rn(v); }

constexpr int SIMT_TILE = 32;  // streamed rows per shared-memory tile

struct SimtParams {
  int NQ, NK, d1, d2, causal;
  float c1, c2;
};

// copy rows [r0, r0+nrows) of a [N][d] matrix into shared memory with row pitch `pitch` floats; rows >= N are zero
template <typename T>
__device__ __forceinline__ void load_rows(float* dst, int pitch, const T* src, int N, int d, int r0, int nrows) {
  for (int idx = threadIdx.x; idx < nrows * d; idx += blockDim.x) {
    const int r = idx / d, k = idx - r * d;
    dst[r * pitch + k] = (r0 + r < N) ? to_f32<T>(src[size_t(r0 + r) * d + k]) : 0.f;
  }
}

// ---------------------------------------------------------------------------------- forward (Alg.1, B_K = 1)
template <typename T>
__global__ void streamkl_fwd_simt_kernel(const T* __restrict__ Q1, const T* __restrict__ K1, const T* __restrict__ Q2,
                                         const T* __restrict__ K2, SimtParams p, float* __restrict__ kl, float* __restrict__ lse1,
                                         float* __restrict__ lse2) {
  extern __shared__ float sm[];
  const int BR = blockDim.x;
  const int p1 = p.d1 + 1, p2 = p.d2 + 1;
  float* sQ1 = sm;                   // [BR][d1+1]
  float* sQ2 = sQ1 + BR * p1;        // [BR][d2+1]
  float* sK1 = sQ2 + BR * p2;        // [TILE][d1]
  float* sK2 = sK1 + SIMT_TILE * p.d1;
  const int bh = blockIdx.y;
  const int q0 = blockIdx.x * BR;
  const T* q1 = Q1 + size_t(bh) * p.NQ * p.d1;
  const T* q2 = Q2 + size_t(bh) * p.NQ * p.d2;
  const T* k1 = K1 + size_t(bh) * p.NK * p.d1;
  const T* k2 = K2 + size_t(bh) * p.NK * p.d2;
  load_rows(sQ1, p1, q1, p.NQ, p.d1, q0, BR);
  load_rows(sQ2, p2, q2, p.NQ, p.d2, q0, BR);
  const int row = q0 + threadIdx.x;
  const int off = p.NK - p.NQ;
  const int limit = p.causal ? min(p.NK - 1, row + off) : p.NK - 1;
  const int blk_limit = p.causal ? min(p.NK - 1, q0 + BR - 1 + off) : p.NK - 1;
  const float L2E = 1.4426950408889634f;
  const float sc1 = p.c1 * L2E, sc2 = p.c2 * L2E;
  float m1 = -CUDART_INF_F, m2 = -CUDART_INF_F, l1 = 0.f, l2 = 0.f, acc = 0.f;
  const float* myq1 = sQ1 + threadIdx.x * p1;
  const float* myq2 = sQ2 + threadIdx.x * p2;
  for (int j0 = 0; j0 <= blk_limit; j0 += SIMT_TILE) {
    __syncthreads();
    load_rows(sK1, p.d1, k1, p.NK, p.d1, j0, SIMT_TILE);
    load_rows(sK2, p.d2, k2, p.NK, p.d2, j0, SIMT_TILE);
    __syncthreads();
    const int jn = min(SIMT_TILE, limit - j0 + 1);
    for (int jj = 0; jj < jn; ++jj) {
      float s1 = 0.f, s2 = 0.f;
      for (int k = 0; k < p.d1; ++k) s1 = fmaf(myq1[k], sK1[jj * p.d1 + k], s1);
      for (int k = 0; k < p.d2; ++k) s2 = fmaf(myq2[k], sK2[jj * p.d2 + k], s2);
      const float x1 = s1 * sc1, x2 = s2 * sc2;  // log2-domain logits
      if (x1 > m1) { const float a = exp2f(m1 - x1); l1 *= a; acc *= a; m1 = x1; }   // Eq.9-10 rescale by alpha1
      if (x2 > m2) { l2 *= exp2f(m2 - x2); m2 = x2; }
      const float e1 = exp2f(x1 - m1);
      l1 += e1;
      l2 += exp2f(x2 - m2);
      acc = fmaf(e1, x1 - x2, acc);
    }
  }
  if (row < p.NQ) {
    const float LN2 = 0.6931471805599453f;
    const float a = LN2 * (m1 + log2f(l1)), b = LN2 * (m2 + log2f(l2));
    const size_t o = size_t(bh) * p.NQ + row;
    lse1[o] = a;
    lse2[o] = b;
    kl[o] = fmaf(LN2, acc / l1, b - a);
  }
}

// ---------------------------------------------------------------------------------- backward
// OWNER_K = false: thread owns query row i, streams key tiles, produces dQ1/dQ2 rows   (Alg.2, Alg.3)
// OWNER_K = true : thread owns key row j,   streams query tiles, produces dK1/dK2 rows
template <typename T, bool OWNER_K>
__global__ void streamkl_bwd_simt_kernel(const T* __restrict__ Q1, const T* __restrict__ K1, const T* __restrict__ Q2,
                                         const T* __restrict__ K2, SimtParams p, const float* __restrict__ kl,
                                         const float* __restrict__ lse1, const float* __restrict__ lse2,
                                         const float* __restrict__ dkl, T* __restrict__ dX1, T* __restrict__ dX2) {
  extern __shared__ float sm[];
  const int BR = blockDim.x;
  const int p1 = p.d1 + 1, p2 = p.d2 + 1;
  float* sX1 = sm;                          // owner rows          [BR][d1+1]
  float* sX2 = sX1 + BR * p1;               //                     [BR][d2+1]
  float* sG1 = sX2 + BR * p2;               // owner gradients     [BR][d1+1]
  float* sG2 = sG1 + BR * p1;               //                     [BR][d2+1]
  float* sY1 = sG2 + BR * p2;               // streamed tile       [TILE][d1]
  float* sY2 = sY1 + SIMT_TILE * p.d1;      //                     [TILE][d2]
  float* sRow = sY2 + SIMT_TILE * p.d2;     // streamed per-query scalars [4][TILE] (OWNER_K only)
  const int bh = blockIdx.y;
  const int NX = OWNER_K ? p.NK : p.NQ, NY = OWNER_K ? p.NQ : p.NK;
  const T* x1 = (OWNER_K ? K1 : Q1) + size_t(bh) * NX * p.d1;
  const T* x2 = (OWNER_K ? K2 : Q2) + size_t(bh) * NX * p.d2;
  const T* y1 = (OWNER_K ? Q1 : K1) + size_t(bh) * NY * p.d1;
  const T* y2 = (OWNER_K ? Q2 : K2) + size_t(bh) * NY * p.d2;
  const float* rkl = kl + size_t(bh) * p.NQ;
  const float* rl1 = lse1 + size_t(bh) * p.NQ;
  const float* rl2 = lse2 + size_t(bh) * p.NQ;
  const float* rg = dkl + size_t(bh) * p.NQ;
  const int x0 = blockIdx.x * BR;
  load_rows(sX1, p1, x1, NX, p.d1, x0, BR);
  load_rows(sX2, p2, x2, NX, p.d2, x0, BR);
  for (int i = threadIdx.x; i < BR * p1; i += BR) sG1[i] = 0.f;
  for (int i = threadIdx.x; i < BR * p2; i += BR) sG2[i] = 0.f;
  const int me = x0 + threadIdx.x;
  const int off = p.NK - p.NQ;
  const float L2E = 1.4426950408889634f;
  const bool teacher = dX1 != nullptr;
  float my_l1 = 0.f, my_l2 = 0.f, my_term = 0.f, my_g = 0.f;
  if (!OWNER_K && me < p.NQ) {
    my_l1 = rl1[me]; my_l2 = rl2[me]; my_g = rg[me];
    my_term = (my_l1 - my_l2) + rkl[me];   // Alg.3: delta + L, subtracted from (s1 - s2)   (Eq.12)
  }
  const float* mx1 = sX1 + threadIdx.x * p1;
  const float* mx2 = sX2 + threadIdx.x * p2;
  float* mg1 = sG1 + threadIdx.x * p1;
  float* mg2 = sG2 + threadIdx.x * p2;
  // range of streamed rows that can interact with this block's owner rows
  int y_begin = 0, y_end = NY;
  if (p.causal) {
    if (OWNER_K) y_begin = max(0, x0 - off);                    // query i sees key j iff j <= i + off
    else         y_end = min(NY, x0 + BR - 1 + off + 1);
  }
  for (int t0 = (y_begin / SIMT_TILE) * SIMT_TILE; t0 < y_end; t0 += SIMT_TILE) {
    __syncthreads();
    load_rows(sY1, p.d1, y1, NY, p.d1, t0, SIMT_TILE);
    load_rows(sY2, p.d2, y2, NY, p.d2, t0, SIMT_TILE);
    if (OWNER_K) {
      for (int i = threadIdx.x; i < SIMT_TILE; i += BR) {
        const int qi = t0 + i;
        const bool ok = qi < p.NQ;
        sRow[i] = ok ? rl1[qi] : 0.f;
        sRow[SIMT_TILE + i] = ok ? rl2[qi] : 0.f;
        sRow[2 * SIMT_TILE + i] = ok ? rg[qi] : 0.f;
        sRow[3 * SIMT_TILE + i] = ok ? (rl1[qi] - rl2[qi]) + rkl[qi] : 0.f;
      }
    }
    __syncthreads();
    if (me >= NX) continue;
    for (int tt = 0; tt < SIMT_TILE; ++tt) {
      const int other = t0 + tt;
      if (other >= NY) break;
      const int qi = OWNER_K ? other : me;
      const int kj = OWNER_K ? me : other;
      if (p.causal && kj > qi + off) { if (OWNER_K) continue; else break; }
      float s1 = 0.f, s2 = 0.f;
      for (int k = 0; k < p.d1; ++k) s1 = fmaf(mx1[k], sY1[tt * p.d1 + k], s1);
      for (int k = 0; k < p.d2; ++k) s2 = fmaf(mx2[k], sY2[tt * p.d2 + k], s2);
      s1 *= p.c1; s2 *= p.c2;
      const float L1 = OWNER_K ? sRow[tt] : my_l1;
      const float L2 = OWNER_K ? sRow[SIMT_TILE + tt] : my_l2;
      const float g = OWNER_K ? sRow[2 * SIMT_TILE + tt] : my_g;
      const float term = OWNER_K ? sRow[3 * SIMT_TILE + tt] : my_term;
      const float P1 = exp2f((s1 - L1) * L2E);       // recompute from saved LSE (Alg.2 line 7)
      const float P2 = exp2f((s2 - L2) * L2E);
      const float ds2 = g * (P2 - P1);               // Alg.2 line 8
      for (int k = 0; k < p.d2; ++k) mg2[k] = fmaf(ds2, sY2[tt * p.d2 + k], mg2[k]);
      if (teacher) {
        const float ds1 = g * P1 * ((s1 - s2) - term);  // Alg.3 lines 9-10
        for (int k = 0; k < p.d1; ++k) mg1[k] = fmaf(ds1, sY1[tt * p.d1 + k], mg1[k]);
      }
    }
  }
  __syncthreads();
  // coalesced write-out, chain-rule factor c_t (R1), one rounding to the output dtype (R13)
  T* o2 = dX2 + size_t(bh) * NX * p.d2;
  for (int idx = threadIdx.x; idx < BR * p.d2; idx += BR) {
    const int r = idx / p.d2, k = idx - r * p.d2;
    if (x0 + r < NX) o2[size_t(x0 + r) * p.d2 + k] = from_f32<T>(p.c2 * sG2[r * p2 + k]);
  }
  if (teacher) {
    T* o1 = dX1 + size_t(bh) * NX * p.d1;
    for (int idx = threadIdx.x; idx < BR * p.d1; idx += BR) {
      const int r = idx / p.d1, k = idx - r * p.d1;
      if (x0 + r < NX) o1[size_t(x0 + r) * p.d1 + k] = from_f32<T>(p.c1 * sG1[r * p1 + k]);
    }
  }
}

}  // namespace skl
