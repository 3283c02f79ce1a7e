// streamkl_bwd_fused.cu -- launcher of the one-visit ("fused") backward kernel and its dQ convert pass; see streamkl.cu for the C ABI.
#include "streamkl_host.cuh"
#include "streamkl_bwd_fused_sm100.cuh"

namespace sklh {
namespace {

skl::OutGeom out_geom(const Strides& st, int d) { return skl::OutGeom{st.b, st.h, st.n, d}; }

// One one-visit pass: zero the fp32 dQ accumulator, run the fused K-owner kernel, convert dQ.
// TPASS = false: student (dS2 -> dQ2, dK2); true: teacher (dS1 -> dQ1, dK1).
template <int D1, int D2, bool CAUSAL, bool TPASS>
int launch_bwd_fused(const void* Q1, const void* K1, const void* Q2, const void* K2, const Shape& s, bool f16, const float4* stats,
                     float* dq_acc, void* dQ, void* dK, cudaStream_t stream) {
  using C = skl::BwdFusedCfg<D1, D2, TPASS>;
  CUtensorMap tm[4];
  if (!make_maps(tm, Q1, K1, Q2, K2, s, C::BY, C::BX, f16)) return STREAMKL_ERR_CUDA;
  auto kern = skl::streamkl_bwd_fused_sm100_kernel<D1, D2, CAUSAL, TPASS>;
  if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES) != cudaSuccess) {
    cudaGetLastError();
    return STREAMKL_ERR_CUDA;
  }
  const size_t n = size_t(s.BH) * s.NQ * C::DG;
  if (cudaMemsetAsync(dq_acc, 0, n * sizeof(float), stream) != cudaSuccess) { cudaGetLastError(); return STREAMKL_ERR_CUDA; }
  skl::BwdFusedParams p;
  p.NQ = s.NQ; p.NK = s.NK; p.BH = int(s.BH);
  p.H = s.H; p.HK = s.HK; p.G = s.G(); p.fmt16 = f16 ? 0u : 1u; p.act2 = s.act2;
  p.TX = (s.NK + C::BX - 1) / C::BX;
  p.c1 = s.c1; p.c2 = s.c2;
  p.stats = stats; p.dq_acc = dq_acc;
  p.dK = static_cast<uint16_t*>(dK);
  p.gk = out_geom(TPASS ? s.k1 : s.k2, TPASS ? s.d1 : s.d2);
  const long long grid = (long long)p.TX * s.B * s.HK;
  if (grid > 0x7fffffffLL) return STREAMKL_ERR_SHAPE;
  {
    ProfScope ps(KID_BWD_FUSED_TC, stream);
    kern<<<dim3((unsigned)grid), C::THREADS, C::SMEM_BYTES, stream>>>(tm[0], tm[1], tm[2], tm[3], p);
  }
  if (cudaGetLastError() != cudaSuccess) return STREAMKL_ERR_CUDA;
  const long long n4 = (long long)(n / 4);
  {
    ProfScope ps(KID_BWD_DQ_CONVERT, stream);
    skl::streamkl_bwd_dq_convert_kernel<<<dim3((unsigned)((n4 + 255) / 256)), 256, 0, stream>>>(
        reinterpret_cast<const float4*>(dq_acc), static_cast<uint16_t*>(dQ), TPASS ? s.c1 * 0.6931471805599453f : s.c2, n4, s.NQ, s.H,
        C::DG, out_geom(TPASS ? s.q1 : s.q2, TPASS ? s.d1 : s.d2), f16 ? 1 : 0);
  }
  if (cudaGetLastError() != cudaSuccess) return STREAMKL_ERR_CUDA;
  g_last_launches += 2;
  return STREAMKL_OK;
}

}  // namespace

int bwd_tc_fused_launch(const void* Q1, const void* K1, const void* Q2, const void* K2, const Shape& s, bool f16, bool teacher_pass,
                        const void* stats_, float* dq_acc, void* dQ, void* dK, cudaStream_t st) {
  const float4* stats = static_cast<const float4*>(stats_);
  const int p1 = pad_dim(s.d1), p2 = pad_dim(s.d2);
#define SKL_FUSED_CASE(A, Bd)                                                                                                      \
  if (p1 == A && p2 == Bd) {                                                                                                       \
    if (teacher_pass) return s.causal ? launch_bwd_fused<A, Bd, true, true>(Q1, K1, Q2, K2, s, f16, stats, dq_acc, dQ, dK, st)     \
                                      : launch_bwd_fused<A, Bd, false, true>(Q1, K1, Q2, K2, s, f16, stats, dq_acc, dQ, dK, st);   \
    return s.causal ? launch_bwd_fused<A, Bd, true, false>(Q1, K1, Q2, K2, s, f16, stats, dq_acc, dQ, dK, st)                      \
                    : launch_bwd_fused<A, Bd, false, false>(Q1, K1, Q2, K2, s, f16, stats, dq_acc, dQ, dK, st);                    \
  }
  SKL_FUSED_CASE(128, 128)
  SKL_FUSED_CASE(128, 64)
  SKL_FUSED_CASE(64, 128)
  SKL_FUSED_CASE(64, 64)
#undef SKL_FUSED_CASE
  return STREAMKL_ERR_SHAPE;
}

}  // namespace sklh
