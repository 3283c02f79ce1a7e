// streamkl.cu -- the C-ABI boundary (include/streamkl.h): argument validation, layouts, strategy selection, the SIMT fallback
// launchers, the host-buffer entry points and profiling.  The tensor-core kernel families are launched through the dispatchers
// of streamkl_host.cuh, each compiled in its own translation unit (streamkl_fwd.cu, streamkl_bwd_q.cu, streamkl_bwd_k.cu,
// streamkl_bwd_fused.cu).  No torch types, no allocation on the device entry points, no CPU fallback.
#include <cuda.h>
#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <cuda_fp16.h>

#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <mutex>
#include <vector>

#include "streamkl_host.cuh"
#include "streamkl_simt.cuh"

namespace sklh {

thread_local int g_last_launches = 0;
thread_local int g_fwd_plan = STREAMKL_FWD_AUTO;

namespace {
struct ProfRecord { int id; cudaEvent_t a, b; };
thread_local bool g_prof_on = false;
thread_local std::vector<ProfRecord>* g_prof = nullptr;
thread_local std::vector<cudaEvent_t>* g_prof_pool = nullptr;   // idle events: created outside the timed region, reused

cudaEvent_t prof_event() {
  if (g_prof_pool && !g_prof_pool->empty()) { cudaEvent_t e = g_prof_pool->back(); g_prof_pool->pop_back(); return e; }
  cudaEvent_t e = nullptr;
  if (cudaEventCreate(&e) != cudaSuccess) { cudaGetLastError(); return nullptr; }
  return e;
}
void prof_release(cudaEvent_t e) {
  if (!e) return;
  if (!g_prof_pool) g_prof_pool = new std::vector<cudaEvent_t>();
  g_prof_pool->push_back(e);
}
}  // namespace

ProfScope::ProfScope(int id, cudaStream_t s) : st(s) {
  if (!g_prof_on) return;
  if (!g_prof) g_prof = new std::vector<ProfRecord>();
  cudaEvent_t a = prof_event();
  if (!a) return;
  b = prof_event();
  if (!b) { prof_release(a); return; }
  cudaEventRecord(a, st);
  g_prof->push_back({id, a, b});
}
ProfScope::~ProfScope() { if (b) cudaEventRecord(b, st); }

namespace {

using EncodeTiledFn = CUresult (*)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                   const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                   CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode_fn() {
  static EncodeTiledFn fn = []() -> EncodeTiledFn {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess)
      return nullptr;
    return reinterpret_cast<EncodeTiledFn>(p);
  }();
  return fn;
}

// true iff the current device is sm_100 (B200): the only target this library is built for
bool device_is_sm100() {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return false; }
  int major = 0;
  if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) { cudaGetLastError(); return false; }
  return major == 10;
}

// 4-D map {d, N, heads, B} of a 16-bit tensor with arbitrary (batch, head, row) strides; box = {64 elements (128 B), box_rows, 1, 1},
// 128-byte swizzle, zero OOB fill: rows beyond N and columns beyond d (head dims that are not 64 / 128) arrive as zeros.
// Encoding a tensor map is a driver call of a microsecond or two, and a backward launches three kernels with four maps each:
// the last few encodings are kept per host thread (a decode-sized split-K forward is ~40 us of GPU time).
struct TmapKey {
  const void* base; int B, heads, N, d, box_rows, f16; long long sb, sh, sn;
  bool operator==(const TmapKey& o) const {
    return base == o.base && B == o.B && heads == o.heads && N == o.N && d == o.d && box_rows == o.box_rows && f16 == o.f16 && sb == o.sb &&
           sh == o.sh && sn == o.sn;
  }
};
struct TmapCache {
  static constexpr int N = 16;
  TmapKey key[N];
  CUtensorMap map[N];
  int used = 0, next = 0;
};
thread_local TmapCache g_tmaps;

bool make_tmap_16(CUtensorMap* m, const void* base, int B, int heads, int N, int d, const Strides& st, int box_rows, bool f16) {
  const TmapKey k{base, B, heads, N, d, box_rows, f16 ? 1 : 0, st.b, st.h, st.n};
  for (int i = 0; i < g_tmaps.used; ++i)
    if (g_tmaps.key[i] == k) { *m = g_tmaps.map[i]; return true; }
  EncodeTiledFn enc = get_encode_fn();
  if (!enc) return false;
  cuuint64_t dims[4] = {cuuint64_t(d), cuuint64_t(N), cuuint64_t(heads), cuuint64_t(B)};
  cuuint64_t strides[3] = {cuuint64_t(st.n) * 2, cuuint64_t(st.h) * 2, cuuint64_t(st.b) * 2};
  cuuint32_t box[4] = {64, cuuint32_t(box_rows), 1, 1};
  cuuint32_t estr[4] = {1, 1, 1, 1};
  if (enc(m, f16 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT16 : CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, const_cast<void*>(base), dims, strides, box,
          estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
    return false;
  const int slot = g_tmaps.used < TmapCache::N ? g_tmaps.used++ : (g_tmaps.next = (g_tmaps.next + 1) % TmapCache::N);
  g_tmaps.key[slot] = k;
  g_tmaps.map[slot] = *m;
  return true;
}

Strides contiguous(int heads, int N, int d) { return Strides{(long long)heads * N * d, (long long)N * d, (long long)d}; }

// fills the layout part of `s` from `L` (NULL = contiguous [B][H][N][d], HK = H) and validates it
int apply_layout(Shape& s, const streamkl_layout* L) {
  s.HK = s.H;
  s.q1 = contiguous(s.H, s.NQ, s.d1); s.k1 = contiguous(s.H, s.NK, s.d1);
  s.q2 = contiguous(s.H, s.NQ, s.d2); s.k2 = contiguous(s.H, s.NK, s.d2);
  s.default_layout = true;
  s.act2 = 0;
  if (!L) return STREAMKL_OK;
  if (L->kv_heads < 0) return STREAMKL_ERR_SHAPE;
  if (L->student_activation != STREAMKL_ACT_NONE && L->student_activation != STREAMKL_ACT_RELU) return STREAMKL_ERR_SHAPE;
  s.act2 = L->student_activation;
  if (L->kv_heads > 0) {
    if (s.H > 0 && (L->kv_heads > s.H || s.H % L->kv_heads != 0)) return STREAMKL_ERR_SHAPE;
    s.HK = L->kv_heads;
    s.k1 = contiguous(s.HK, s.NK, s.d1); s.k2 = contiguous(s.HK, s.NK, s.d2);
  }
  auto take = [&](const long long (&v)[3], Strides& dst, int d, int N) -> int {
    if (v[0] == 0 && v[1] == 0 && v[2] == 0) return STREAMKL_OK;          // default for this tensor
    if (v[0] < 0 || v[1] < 0 || v[2] < d) return STREAMKL_ERR_SHAPE;       // rows must not overlap; broadcast batch / head (0) is allowed
    if ((v[0] | v[1] | v[2]) & 7) return STREAMKL_ERR_ALIGN;               // 16-byte multiples (TMA global strides)
    (void)N;
    dst = Strides{v[0], v[1], v[2]};
    return STREAMKL_OK;
  };
  int rc;
  if ((rc = take(L->q1_stride, s.q1, s.d1, s.NQ)) != STREAMKL_OK || (rc = take(L->k1_stride, s.k1, s.d1, s.NK)) != STREAMKL_OK ||
      (rc = take(L->q2_stride, s.q2, s.d2, s.NQ)) != STREAMKL_OK || (rc = take(L->k2_stride, s.k2, s.d2, s.NK)) != STREAMKL_OK)
    return rc;
  auto same = [](const Strides& a, const Strides& b) { return a.b == b.b && a.h == b.h && a.n == b.n; };
  s.default_layout = s.act2 == 0 && s.HK == s.H && same(s.q1, contiguous(s.H, s.NQ, s.d1)) && same(s.k1, contiguous(s.H, s.NK, s.d1)) &&
                     same(s.q2, contiguous(s.H, s.NQ, s.d2)) && same(s.k2, contiguous(s.H, s.NK, s.d2));
  return STREAMKL_OK;
}

// true iff the [B][heads][N][d] view with these element strides maps distinct (b, h, n) to disjoint d-element rows.  The test is
// the nested one -- dimensions of extent > 1 taken by growing stride, each stride at least the span of everything below it -- so
// broadcast dimensions (stride 0 with extent > 1), head strides below d and interleavings that fold onto themselves fail it.
// Gradients are written with their input's strides by one owner CTA per tile: on a view that overlaps itself several owners
// would store to the same addresses and the last one would win where the true gradient is the sum.
bool rows_are_disjoint(const Strides& st, long long B, long long heads, long long N, int d) {
  long long sv[3] = {st.b, st.h, st.n}, ev[3] = {B, heads, N};
  for (int i = 0; i < 3; ++i)
    for (int j = i + 1; j < 3; ++j)
      if (sv[j] < sv[i]) { std::swap(sv[i], sv[j]); std::swap(ev[i], ev[j]); }
  long long span = d;
  for (int i = 0; i < 3; ++i) {
    if (ev[i] <= 1) continue;
    if (sv[i] < span) return false;
    if (sv[i] > (1LL << 46) / ev[i]) return false;   // (also keeps span inside 64 bits; validate_common bounds the extents)
    span += sv[i] * (ev[i] - 1);
  }
  return true;
}

int validate_common(const void* Q1, const void* K1, const void* Q2, const void* K2, const Shape& s) {
  if (s.B < 0 || s.H < 0 || s.NQ < 0 || s.NK < 1 || s.d1 < 1 || s.d2 < 1 || s.d1 > 256 || s.d2 > 256) return STREAMKL_ERR_SHAPE;
  if (s.causal && s.NQ > s.NK) return STREAMKL_ERR_SHAPE;
  if (s.BH > 65535 * 1024LL || s.BH * (long long)(s.NQ > s.NK ? s.NQ : s.NK) > (1LL << 40)) return STREAMKL_ERR_SHAPE;
  if (!(std::isfinite(s.c1) && std::isfinite(s.c2) && s.c1 > 0.f && s.c2 > 0.f)) return STREAMKL_ERR_SCALE;
  if (s.BH == 0 || s.NQ == 0) return STREAMKL_OK;
  if (!Q1 || !K1 || !Q2 || !K2) return STREAMKL_ERR_NULLPTR;
  if ((reinterpret_cast<uintptr_t>(Q1) | reinterpret_cast<uintptr_t>(K1) | reinterpret_cast<uintptr_t>(Q2) |
       reinterpret_cast<uintptr_t>(K2)) & 15)
    return STREAMKL_ERR_ALIGN;
  return STREAMKL_OK;
}

// tensor-core path: 16-bit inputs, head dims that are multiples of 8 (TMA: 16-byte rows) up to 256.  The kernels work on
// head dims zero-padded to the next multiple of 64 (pad_dim): fixed plans for {64,128}^2, run-time K-block counts when a
// head dim exceeds 128 (wide_dims).
bool tc_dims(int d1, int d2) { return d1 % 8 == 0 && d2 % 8 == 0 && d1 >= 8 && d2 >= 8 && d1 <= kMaxTcDim && d2 <= kMaxTcDim; }
bool tc_shape(int dtype, const Shape& s) { return (dtype == STREAMKL_BF16 || dtype == STREAMKL_F16) && tc_dims(s.d1, s.d2); }

}  // namespace

bool make_maps(CUtensorMap (&t)[4], const void* Q1, const void* K1, const void* Q2, const void* K2, const Shape& s, int rows_q, int rows_k,
               bool f16) {
  return make_tmap_16(&t[0], Q1, s.B, s.H, s.NQ, s.d1, s.q1, rows_q, f16) && make_tmap_16(&t[1], K1, s.B, s.HK, s.NK, s.d1, s.k1, rows_k, f16) &&
         make_tmap_16(&t[2], Q2, s.B, s.H, s.NQ, s.d2, s.q2, rows_q, f16) && make_tmap_16(&t[3], K2, s.B, s.HK, s.NK, s.d2, s.k2, rows_k, f16);
}

}  // namespace sklh

namespace {
using namespace sklh;

thread_local int g_bwd_mode = STREAMKL_BWD_AUTO;

// ---- optional per-kernel timing (streamkl_profile_*): CUDA events recorded on the launch stream around every kernel
const char* const kKernelNames[KID_COUNT] = {"streamkl_fwd_sm100_kernel", "streamkl_bwd_sm100_kernel<OWNER_Q>",
                                             "streamkl_bwd_sm100_kernel<OWNER_K>", "streamkl_fwd_simt_kernel",
                                             "streamkl_bwd_simt_kernel<OWNER_Q>", "streamkl_bwd_simt_kernel<OWNER_K>",
                                             "streamkl_bwd_stats_kernel", "streamkl_fwd_sm100_kernel<SPLIT>",
                                             "streamkl_fwd_splitk_reduce_kernel", "streamkl_bwd_fused_sm100_kernel",
                                             "streamkl_bwd_dq_convert_kernel", "streamkl_bwd_wide_sm100_kernel<OWNER_Q>",
                                             "streamkl_bwd_wide_sm100_kernel<OWNER_K>"};
// ----------------------------------------------------------------------------------------- forward (SIMT fallback, dispatch)
int simt_block_rows(size_t floats_per_row, size_t fixed_floats, size_t* smem_bytes) {
  for (int br : {128, 64, 32}) {
    size_t b = (floats_per_row * br + fixed_floats) * sizeof(float);
    if (b <= 200 * 1024) { *smem_bytes = b; return br; }
  }
  return 0;
}

template <typename T>
int launch_fwd_simt(const void* Q1, const void* K1, const void* Q2, const void* K2, const Shape& s, float* kl, float* lse1,
                    float* lse2, cudaStream_t stream) {
  size_t smem = 0;
  const int br = simt_block_rows(size_t(s.d1 + s.d2 + 2), size_t(skl::SIMT_TILE) * (s.d1 + s.d2), &smem);
  if (!br) return STREAMKL_ERR_SHAPE;
  auto kern = skl::streamkl_fwd_simt_kernel<T>;
  if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, int(smem)) != cudaSuccess) {
    cudaGetLastError();
    return STREAMKL_ERR_CUDA;
  }
  skl::SimtParams p{s.NQ, s.NK, s.d1, s.d2, s.causal, s.c1, s.c2};
  dim3 grid((s.NQ + br - 1) / br, (unsigned)s.BH);
  {
    ProfScope ps(KID_FWD_SIMT, stream);
    kern<<<grid, br, smem, stream>>>(static_cast<const T*>(Q1), static_cast<const T*>(K1), static_cast<const T*>(Q2),
                                     static_cast<const T*>(K2), p, kl, lse1, lse2);
  }
  if (cudaGetLastError() != cudaSuccess) return STREAMKL_ERR_CUDA;
  g_last_launches += 1;
  return STREAMKL_OK;
}

int fwd_dispatch(int dtype, const streamkl_layout* L, const void* Q1, const void* K1, const void* Q2, const void* K2, int B, int H, int NQ,
                 int NK, int d1, int d2, float c1, float c2, int causal, float* kl, float* lse1, float* lse2, cudaStream_t stream,
                 int splits = 1, float* part = nullptr) {
  if (dtype != STREAMKL_BF16 && dtype != STREAMKL_F16 && dtype != STREAMKL_F32) return STREAMKL_ERR_DTYPE;
  Shape s{B, H, NQ, NK, d1, d2, causal ? 1 : 0, c1, c2, (long long)B * (long long)H};
  int rc = validate_common(Q1, K1, Q2, K2, s);
  if (rc != STREAMKL_OK) return rc;
  if ((rc = apply_layout(s, L)) != STREAMKL_OK) return rc;
  g_last_launches = 0;
  if (s.BH == 0 || s.NQ == 0) return STREAMKL_OK;
  if (!kl || !lse1 || !lse2) return STREAMKL_ERR_NULLPTR;
  if (!tc_shape(dtype, s) && !s.default_layout) return STREAMKL_ERR_SHAPE;   // strides / shared K heads: tensor-core path only
  if (!device_is_sm100()) return STREAMKL_ERR_CUDA;
  if (tc_shape(dtype, s)) return fwd_tc_launch(Q1, K1, Q2, K2, s, dtype == STREAMKL_F16, kl, lse1, lse2, stream, splits, part);
  if (s.BH > 65535) return STREAMKL_ERR_SHAPE;   // SIMT grids put the head index in gridDim.y
  if (dtype == STREAMKL_BF16) return launch_fwd_simt<__nv_bfloat16>(Q1, K1, Q2, K2, s, kl, lse1, lse2, stream);
  if (dtype == STREAMKL_F16) return launch_fwd_simt<__half>(Q1, K1, Q2, K2, s, kl, lse1, lse2, stream);
  return launch_fwd_simt<float>(Q1, K1, Q2, K2, s, kl, lse1, lse2, stream);
}

// ----------------------------------------------------------------------------------------- backward (SIMT fallback, strategy, dispatch)
template <typename T, bool OWNER_K>
int launch_bwd_simt(const void* Q1, const void* K1, const void* Q2, const void* K2, const Shape& s, const float* kl,
                    const float* lse1, const float* lse2, const float* dkl, void* dX1, void* dX2, cudaStream_t stream) {
  size_t smem = 0;
  const int br = simt_block_rows(size_t(2 * (s.d1 + s.d2 + 2)), size_t(skl::SIMT_TILE) * (s.d1 + s.d2 + 4), &smem);
  if (!br) return STREAMKL_ERR_SHAPE;
  auto kern = skl::streamkl_bwd_simt_kernel<T, OWNER_K>;
  if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, int(smem)) != cudaSuccess) {
    cudaGetLastError();
    return STREAMKL_ERR_CUDA;
  }
  skl::SimtParams p{s.NQ, s.NK, s.d1, s.d2, s.causal, s.c1, s.c2};
  const int NX = OWNER_K ? s.NK : s.NQ;
  dim3 grid((NX + br - 1) / br, (unsigned)s.BH);
  {
    ProfScope ps(OWNER_K ? KID_BWD_DK_SIMT : KID_BWD_DQ_SIMT, stream);
    kern<<<grid, br, smem, stream>>>(static_cast<const T*>(Q1), static_cast<const T*>(K1), static_cast<const T*>(Q2),
                                     static_cast<const T*>(K2), p, kl, lse1, lse2, dkl, static_cast<T*>(dX1), static_cast<T*>(dX2));
  }
  if (cudaGetLastError() != cudaSuccess) return STREAMKL_ERR_CUDA;
  g_last_launches += 1;
  return STREAMKL_OK;
}

// Strategy selection of the backward (see bwd_tc_both): the one-visit kernels iff the mode is FUSED, or AUTO below the measured
// crossover (bench.py "backward strategies", profiles/r02_bwd_strategies.md): at most four 128-query tiles per head for
// Setting 1 (one pass: half the recomputation), at most two for Setting 2 (two passes: same work as the owner kernels, the
// gain is the fuller K-owner grid).  streamkl_bwd_workspace_bytes applies the same rule, so the fp32 dQ accumulators are
// only asked for when the strategy that will run needs them.
bool bwd_fused_selected(int NQ, bool teacher, int d1, int d2) {
  if (wide_dims(d1, d2)) return false;   // head dims above 128: owner kernels only (TMEM has no room for the dQ^T stages)
  if (g_bwd_mode == STREAMKL_BWD_FUSED) return true;
  if (g_bwd_mode != STREAMKL_BWD_AUTO) return false;
  if ((NQ + 127) / 128 <= (teacher ? 2 : 4)) return true;   // small N_Q: the Q-owner grid is too small to fill the GPU
  // Setting 1 with a narrow student at long context (the indexer case): the owner kernels pay two recomputations and four exps per
  // pair for 2 d2 gradient MACs, the one-visit pass pays one and two.  Measured (profiles/r03_bwd_strategies_large.md, both run orders):
  // d2 = 64, N >= 32K: one-visit 7-11 % faster (causal 10-11 %, unmasked 7.3-7.6 %); N = 16K: a tie; d2 = 128: within +-4 % everywhere.
  return !teacher && pad_dim(d2) <= 64 && NQ >= 32768;
}
size_t fused_acc_bytes_aligned(long long BH, int NQ, int d) { return (size_t(BH) * size_t(NQ) * size_t(d) * sizeof(float) + 255) & ~size_t(255); }

size_t stats_bytes_aligned(long long BH, int NQ) { return (size_t(BH) * size_t(stats_padded_rows(NQ)) * 16 + 255) & ~size_t(255); }

// B1 pre-pass, then the selected strategy.
int bwd_tc_both(const void* Q1, const void* K1, const void* Q2, const void* K2, const Shape& s, bool f16, const float* kl, const float* lse1,
                const float* lse2, const float* dkl, void* dQ1, void* dK1, void* dQ2, void* dK2, void* workspace, cudaStream_t st) {
  const bool t = dQ1 != nullptr;
  int rc = bwd_stats_launch(s, kl, lse1, lse2, dkl, workspace, st);
  if (rc != STREAMKL_OK) return rc;
  // Strategy (PAPER.md:321 picks fused iff T_Q*C <= T_K with an empirically tuned C).  Measured on B200
  // (profiles/r01f_fused_bwd.md, r02_bwd_strategies.md): the one-visit kernels win while the Q-owner grid is small (Setting 1:
  // 1.3-3.0x up to T_Q = 4 tiles of 128 queries, level at 8; Setting 2: 1.3-1.5x up to T_Q = 2, 0.8x at 4) and lose beyond,
  // where their fp32 atomics (64 KB per 128x128 tile pair and pass) run into the L2's atomic throughput; the crossover did
  // not move with T_K (128 vs 1024), so the rule is on T_Q alone.
  if (bwd_fused_selected(s.NQ, t, s.d1, s.d2)) {   // one visit per differentiated distribution, dQ through fp32 atomics
    uint8_t* w = static_cast<uint8_t*>(workspace) + stats_bytes_aligned(s.BH, s.NQ);
    float* acc2 = reinterpret_cast<float*>(w);
    float* acc1 = reinterpret_cast<float*>(w + fused_acc_bytes_aligned(s.BH, s.NQ, pad_dim(s.d2)));
    rc = bwd_tc_fused_launch(Q1, K1, Q2, K2, s, f16, false, workspace, acc2, dQ2, dK2, st);
    if (rc != STREAMKL_OK || !t) return rc;
    return bwd_tc_fused_launch(Q1, K1, Q2, K2, s, f16, true, workspace, acc1, dQ1, dK1, st);
  }
  if (wide_dims(s.d1, s.d2)) {
    rc = bwd_wide_owner_q_launch(Q1, K1, Q2, K2, s, f16, workspace, dQ1, dQ2, st);
    if (rc != STREAMKL_OK) return rc;
    return bwd_wide_owner_k_launch(Q1, K1, Q2, K2, s, f16, workspace, dK1, dK2, st);
  }
  rc = bwd_tc_owner_q_launch(Q1, K1, Q2, K2, s, f16, workspace, dQ1, dQ2, st);
  if (rc != STREAMKL_OK) return rc;
  return bwd_tc_owner_k_launch(Q1, K1, Q2, K2, s, f16, workspace, dK1, dK2, st);
}

int bwd_dispatch(int dtype, const streamkl_layout* L, const void* Q1, const void* K1, const void* Q2, const void* K2, int B, int H, int NQ,
                 int NK, int d1, int d2, float c1, float c2, int causal, const float* kl, const float* lse1, const float* lse2,
                 const float* dkl, void* dQ1, void* dK1, void* dQ2, void* dK2, void* workspace, size_t workspace_bytes, cudaStream_t stream) {
  if (dtype != STREAMKL_BF16 && dtype != STREAMKL_F16 && dtype != STREAMKL_F32) return STREAMKL_ERR_DTYPE;
  Shape s{B, H, NQ, NK, d1, d2, causal ? 1 : 0, c1, c2, (long long)B * (long long)H};
  int rc = validate_common(Q1, K1, Q2, K2, s);
  if (rc != STREAMKL_OK) return rc;
  if ((rc = apply_layout(s, L)) != STREAMKL_OK) return rc;
  g_last_launches = 0;
  if ((dQ1 == nullptr) != (dK1 == nullptr)) return STREAMKL_ERR_NULLPTR;
  // the forward may read broadcast or overlapping views; the backward writes dX through the same strides, so every view that
  // receives a gradient must address disjoint rows
  if (!rows_are_disjoint(s.q2, s.B, s.H, s.NQ, s.d2) || !rows_are_disjoint(s.k2, s.B, s.HK, s.NK, s.d2)) return STREAMKL_ERR_SHAPE;
  if (dQ1 && dK1 && (!rows_are_disjoint(s.q1, s.B, s.H, s.NQ, s.d1) || !rows_are_disjoint(s.k1, s.B, s.HK, s.NK, s.d1)))
    return STREAMKL_ERR_SHAPE;
  if (s.BH == 0) return STREAMKL_OK;
  if (!dK2) return STREAMKL_ERR_NULLPTR;
  if (s.NQ > 0 && (!kl || !lse1 || !lse2 || !dkl || !dQ2)) return STREAMKL_ERR_NULLPTR;
  if ((reinterpret_cast<uintptr_t>(dQ1) | reinterpret_cast<uintptr_t>(dK1) | reinterpret_cast<uintptr_t>(dQ2) |
       reinterpret_cast<uintptr_t>(dK2)) & 15)
    return STREAMKL_ERR_ALIGN;
  const size_t need = streamkl_bwd_workspace_bytes(B, H, NQ, NK, d1, d2, dQ1 != nullptr);
  if (need > 0 && (!workspace || workspace_bytes < need)) return STREAMKL_ERR_WORKSPACE;
  if (reinterpret_cast<uintptr_t>(workspace) & 15) return STREAMKL_ERR_ALIGN;
  if (!tc_shape(dtype, s) && !s.default_layout) return STREAMKL_ERR_SHAPE;   // strides / shared K heads: tensor-core path only
  if (!device_is_sm100()) return STREAMKL_ERR_CUDA;
  const size_t es = dtype == STREAMKL_F32 ? 4 : 2;
  if (s.NQ == 0) {  // no query rows: dK = 0, nothing else to write
    if (!s.default_layout) return STREAMKL_ERR_SHAPE;
    if (cudaMemsetAsync(dK2, 0, size_t(s.BH) * NK * d2 * es, stream) != cudaSuccess) return STREAMKL_ERR_CUDA;
    if (dK1 && cudaMemsetAsync(dK1, 0, size_t(s.BH) * NK * d1 * es, stream) != cudaSuccess) return STREAMKL_ERR_CUDA;
    return STREAMKL_OK;
  }
  if (tc_shape(dtype, s))
    return bwd_tc_both(Q1, K1, Q2, K2, s, dtype == STREAMKL_F16, kl, lse1, lse2, dkl, dQ1, dK1, dQ2, dK2, workspace, stream);
  if (s.BH > 65535) return STREAMKL_ERR_SHAPE;   // SIMT grids put the head index in gridDim.y
  if (dtype == STREAMKL_BF16) {
    rc = launch_bwd_simt<__nv_bfloat16, false>(Q1, K1, Q2, K2, s, kl, lse1, lse2, dkl, dQ1, dQ2, stream);
    if (rc != STREAMKL_OK) return rc;
    return launch_bwd_simt<__nv_bfloat16, true>(Q1, K1, Q2, K2, s, kl, lse1, lse2, dkl, dK1, dK2, stream);
  }
  if (dtype == STREAMKL_F16) {
    rc = launch_bwd_simt<__half, false>(Q1, K1, Q2, K2, s, kl, lse1, lse2, dkl, dQ1, dQ2, stream);
    if (rc != STREAMKL_OK) return rc;
    return launch_bwd_simt<__half, true>(Q1, K1, Q2, K2, s, kl, lse1, lse2, dkl, dK1, dK2, stream);
  }
  rc = launch_bwd_simt<float, false>(Q1, K1, Q2, K2, s, kl, lse1, lse2, dkl, dQ1, dQ2, stream);
  if (rc != STREAMKL_OK) return rc;
  return launch_bwd_simt<float, true>(Q1, K1, Q2, K2, s, kl, lse1, lse2, dkl, dK1, dK2, stream);
}

// Device scratch of the *_host entry points, taken from the device's stream-ordered pool.  The pool keeps freed blocks
// (release threshold = max), so a host call after the first one pays no cudaMalloc / cudaFree; streamkl_host_trim()
// hands the memory back to the driver.
struct AsyncScratch {
  cudaStream_t st;
  std::vector<void*> ptrs;
  bool ok = true;
  explicit AsyncScratch(cudaStream_t s) : st(s) {
    int dev = 0;
    cudaMemPool_t pool;
    if (cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetDefaultMemPool(&pool, dev) == cudaSuccess) {
      unsigned long long thr = ~0ull;
      cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &thr);
    }
    cudaGetLastError();
  }
  void* get(size_t n) {
    if (n == 0) return nullptr;
    void* p = nullptr;
    if (cudaMallocAsync(&p, n, st) != cudaSuccess) { cudaGetLastError(); ok = false; return nullptr; }
    ptrs.push_back(p);
    return p;
  }
  ~AsyncScratch() {
    for (void* p : ptrs) cudaFreeAsync(p, st);
    cudaStreamSynchronize(st);
  }
};

// Two helper streams per host thread: uploads and downloads of one head group overlap the kernels of another.
struct HostStreams {
  cudaStream_t in = nullptr, out = nullptr, cmp = nullptr;
  bool ok = false;
  HostStreams() {
    ok = cudaStreamCreateWithFlags(&in, cudaStreamNonBlocking) == cudaSuccess &&
         cudaStreamCreateWithFlags(&out, cudaStreamNonBlocking) == cudaSuccess &&
         cudaStreamCreateWithFlags(&cmp, cudaStreamNonBlocking) == cudaSuccess;
    if (!ok) cudaGetLastError();
  }
  ~HostStreams() {   // the owning host thread ends: give the helper streams back (ignore errors at process teardown)
    if (in) cudaStreamDestroy(in);
    if (out) cudaStreamDestroy(out);
    if (cmp) cudaStreamDestroy(cmp);
    cudaGetLastError();
  }
};
HostStreams& host_streams() {
  thread_local HostStreams hs;
  return hs;
}

// ---- streamkl_fwd_splitk_noalloc: split-K partials in memory that is part of the loaded library image
// The array below is reserved on every GPU this process uses the library on, from the moment the CUDA module is loaded there until
// the process exits.  Host code must never hand the NAME of the array to a kernel: on the host that name is only a handle for the
// runtime's symbol table (a kernel given it would fault or, on systems where the GPU can read host memory, quietly use the wrong
// bytes).  The real device address is asked for once per device, with that device current, and remembered.
constexpr size_t kNoAllocScratchBytes = size_t(STREAMKL_NOALLOC_SCRATCH_BYTES);
static __device__ __align__(256) unsigned char g_noalloc_scratch[kNoAllocScratchBytes];

constexpr int kNoAllocMaxDevices = 64;
std::atomic<float*> g_noalloc_addr[kNoAllocMaxDevices];   // zero-initialised: "not looked up yet" for that device ordinal
std::mutex g_noalloc_mutex;

// Device address of g_noalloc_scratch on the CURRENT device (looked up on the first call per device, then cached).
int noalloc_scratch_on_current_device(float** out) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kNoAllocMaxDevices) { cudaGetLastError(); return STREAMKL_ERR_CUDA; }
  float* p = g_noalloc_addr[dev].load(std::memory_order_acquire);
  if (!p) {
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    p = g_noalloc_addr[dev].load(std::memory_order_relaxed);
    if (!p) {
      void* q = nullptr;
      if (cudaGetSymbolAddress(&q, g_noalloc_scratch) != cudaSuccess || !q) { cudaGetLastError(); return STREAMKL_ERR_CUDA; }
      p = static_cast<float*>(q);
      g_noalloc_addr[dev].store(p, std::memory_order_release);
    }
  }
  *out = p;
  return STREAMKL_OK;
}

}  // namespace

extern "C" {

int streamkl_fwd(const void* Q1, const void* K1, const void* Q2, const void* K2, int B, int H, int NQ, int NK, int d1, int d2, float c1,
                 float c2, int causal, float* kl_rows, float* lse1, float* lse2, streamkl_stream_t stream) {
  return fwd_dispatch(STREAMKL_BF16, nullptr, Q1, K1, Q2, K2, B, H, NQ, NK, d1, d2, c1, c2, causal, kl_rows, lse1, lse2,
                      static_cast<cudaStream_t>(stream));
}
int streamkl_fwd_f32(const void* Q1, const void* K1, const void* Q2, const void* K2, int B, int H, int NQ, int NK, int d1, int d2,
                     float c1, float c2, int causal, float* kl_rows, float* lse1, float* lse2, streamkl_stream_t stream) {
  return fwd_dispatch(STREAMKL_F32, nullptr, Q1, K1, Q2, K2, B, H, NQ, NK, d1, d2, c1, c2, causal, kl_rows, lse1, lse2,
                      static_cast<cudaStream_t>(stream));
}
int streamkl_bwd(const void* Q1, const void* K1, const void* Q2, const void* K2, int B, int H, int NQ, int NK, int d1, int d2, float c1,
                 float c2, int causal, const float* kl_rows, const float* lse1, const float* lse2, const float* dkl_rows, void* dQ1,
                 void* dK1, void* dQ2, void* dK2, void* workspace, size_t workspace_bytes, streamkl_stream_t stream) {
  return bwd_dispatch(STREAMKL_BF16, nullptr, Q1, K1, Q2, K2, B, H, NQ, NK, d1, d2, c1, c2, causal, kl_rows, lse1, lse2, dkl_rows, dQ1, dK1,
                      dQ2, dK2, workspace, workspace_bytes, static_cast<cudaStream_t>(stream));
}
int streamkl_bwd_f32(const void* Q1, const void* K1, const void* Q2, const void* K2, int B, int H, int NQ, int NK, int d1, int d2,
                     float c1, float c2, int causal, const float* kl_rows, const float* lse1, const float* lse2,
                     const float* dkl_rows, void* dQ1, void* dK1, void* dQ2, void* dK2, void* workspace, size_t workspace_bytes,
                     streamkl_stream_t stream) {
  return bwd_dispatch(STREAMKL_F32, nullptr, Q1, K1, Q2, K2, B, H, NQ, NK, d1, d2, c1, c2, causal, kl_rows, lse1, lse2, dkl_rows, dQ1, dK1,
                      dQ2, dK2, workspace, workspace_bytes, static_cast<cudaStream_t>(stream));
}

int streamkl_fwd_ex(const streamkl_layout* layout, const void* Q1, const void* K1, const void* Q2, const void* K2, int B, int H, int NQ, int NK,
                    int d1, int d2, float c1, float c2, int causal, float* kl_rows, float* lse1, float* lse2, streamkl_stream_t stream) {
  return fwd_dispatch(layout ? layout->dtype : STREAMKL_BF16, layout, Q1, K1, Q2, K2, B, H, NQ, NK, d1, d2, c1, c2, causal, kl_rows, lse1, lse2,
                      static_cast<cudaStream_t>(stream));
}
int streamkl_bwd_ex(const streamkl_layout* layout, const void* Q1, const void* K1, const void* Q2, const void* K2, int B, int H, int NQ, int NK,
                    int d1, int d2, float c1, float c2, int causal, const float* kl_rows, const float* lse1, const float* lse2,
                    const float* dkl_rows, void* dQ1, void* dK1, void* dQ2, void* dK2, void* workspace, size_t workspace_bytes,
                    streamkl_stream_t stream) {
  return bwd_dispatch(layout ? layout->dtype : STREAMKL_BF16, layout, Q1, K1, Q2, K2, B, H, NQ, NK, d1, d2, c1, c2, causal, kl_rows, lse1, lse2,
                      dkl_rows, dQ1, dK1, dQ2, dK2, workspace, workspace_bytes, static_cast<cudaStream_t>(stream));
}

int streamkl_fwd_splitk_splits(int B, int H, int NQ, int NK, int p_target) {
  // adaptive split selection: P_base = bsz * T_Q; W = 1 if P_base >= P_target, else min(floor(P_target / P_base), T_K)
  if (B <= 0 || H <= 0 || NQ <= 0 || NK <= 0) return 1;
  if (p_target <= 0) p_target = 148;   // one CTA per SM of a B200 = one full wave (measured best: profiles/r01d_splitk.md)
  const long long p_base = (long long)B * H * ((NQ + kFwdBQ - 1) / kFwdBQ);
  const long long tk = (NK + kFwdBK - 1) / kFwdBK;
  if (p_base >= p_target) return 1;
  const long long w = p_target / p_base;
  return int(w < tk ? w : tk);
}

size_t streamkl_fwd_splitk_workspace_bytes(int B, int H, int NQ, int splits) {
  if (B <= 0 || H <= 0 || NQ <= 0 || splits <= 1) return 0;
  return size_t(B) * size_t(H) * size_t(splits) * 5 * size_t(NQ) * sizeof(float);
}

int streamkl_fwd_splitk_ex(const streamkl_layout* layout, const void* Q1, const void* K1, const void* Q2, const void* K2, int B, int H, int NQ,
                           int NK, int d1, int d2, float c1, float c2, int causal, int splits, float* kl_rows, float* lse1, float* lse2,
                           void* workspace, size_t workspace_bytes, streamkl_stream_t stream) {
  const int dtype = layout ? layout->dtype : STREAMKL_BF16;
  if (splits <= 0) splits = streamkl_fwd_splitk_splits(B, H, NQ, NK, 0);
  const int tk = NK > 0 ? (NK + kFwdBK - 1) / kFwdBK : 1;
  if (splits > tk) splits = tk;
  const bool tc = tc_dims(d1, d2) && (dtype == STREAMKL_BF16 || dtype == STREAMKL_F16);
  if (!tc || splits <= 1)   // other head dims / fp32 run the (unsplit) SIMT kernel; W = 1 is the default kernel
    return fwd_dispatch(dtype, layout, Q1, K1, Q2, K2, B, H, NQ, NK, d1, d2, c1, c2, causal, kl_rows, lse1, lse2,
                        static_cast<cudaStream_t>(stream));
  const size_t need = streamkl_fwd_splitk_workspace_bytes(B, H, NQ, splits);
  if (need > 0 && (!workspace || workspace_bytes < need)) return STREAMKL_ERR_WORKSPACE;
  if (reinterpret_cast<uintptr_t>(workspace) & 15) return STREAMKL_ERR_ALIGN;
  return fwd_dispatch(dtype, layout, Q1, K1, Q2, K2, B, H, NQ, NK, d1, d2, c1, c2, causal, kl_rows, lse1, lse2,
                      static_cast<cudaStream_t>(stream), splits, static_cast<float*>(workspace));
}

int streamkl_fwd_splitk(const void* Q1, const void* K1, const void* Q2, const void* K2, int B, int H, int NQ, int NK, int d1, int d2,
                        float c1, float c2, int causal, int splits, float* kl_rows, float* lse1, float* lse2, void* workspace,
                        size_t workspace_bytes, streamkl_stream_t stream) {
  return streamkl_fwd_splitk_ex(nullptr, Q1, K1, Q2, K2, B, H, NQ, NK, d1, d2, c1, c2, causal, splits, kl_rows, lse1, lse2, workspace,
                                workspace_bytes, stream);
}

size_t streamkl_fwd_splitk_noalloc_capacity(void) { return kNoAllocScratchBytes; }

int streamkl_fwd_splitk_noalloc(const void* Q1, const void* K1, const void* Q2, const void* K2, int B, int H, int NQ, int NK, int d1, int d2,
                                float c1, float c2, int causal, int splits, float* kl_rows, float* lse1, float* lse2,
                                streamkl_stream_t stream) {
  const bool adaptive = splits <= 0;
  if (adaptive) splits = streamkl_fwd_splitk_splits(B, H, NQ, NK, 0);
  const int tk = NK > 0 ? (NK + kFwdBK - 1) / kFwdBK : 1;
  if (splits > tk) splits = tk;
  // an adaptive W is lowered until its partials fit the built-in scratch (W = 1 needs none); an explicit W that does not fit is refused
  while (adaptive && splits > 1 && streamkl_fwd_splitk_workspace_bytes(B, H, NQ, splits) > kNoAllocScratchBytes) --splits;
  if (!tc_dims(d1, d2) || splits <= 1)   // unsplit kernels: they write nothing but the outputs, so there is no scratch to provide
    return fwd_dispatch(STREAMKL_BF16, nullptr, Q1, K1, Q2, K2, B, H, NQ, NK, d1, d2, c1, c2, causal, kl_rows, lse1, lse2,
                        static_cast<cudaStream_t>(stream));
  if (streamkl_fwd_splitk_workspace_bytes(B, H, NQ, splits) > kNoAllocScratchBytes) return STREAMKL_ERR_SCRATCH_LIMIT;
  // argument errors are reported before the device is touched (the same checks fwd_dispatch repeats below)
  Shape s{B, H, NQ, NK, d1, d2, causal ? 1 : 0, c1, c2, (long long)B * (long long)H};
  int rc = validate_common(Q1, K1, Q2, K2, s);
  if (rc != STREAMKL_OK) return rc;
  if (s.BH == 0 || s.NQ == 0) return STREAMKL_OK;
  if (!kl_rows || !lse1 || !lse2) return STREAMKL_ERR_NULLPTR;
  if (!device_is_sm100()) return STREAMKL_ERR_CUDA;
  float* part = nullptr;
  if ((rc = noalloc_scratch_on_current_device(&part)) != STREAMKL_OK) return rc;
  // Nothing has to be cleared: the split kernel stores all five statistics of every (head, chunk, row) slot the reduce kernel
  // reads -- identity values for chunks a causal row cannot see -- so what an earlier call left in the array is never read.
  return fwd_dispatch(STREAMKL_BF16, nullptr, Q1, K1, Q2, K2, B, H, NQ, NK, d1, d2, c1, c2, causal, kl_rows, lse1, lse2,
                      static_cast<cudaStream_t>(stream), splits, part);
}

size_t streamkl_bwd_workspace_bytes(int B, int H, int NQ, int, int d1, int d2, int want_teacher) {
  // both gradients are produced by tile ownership: no fp32 accumulation workspace.  The tcgen05 kernels read the
  // per-query scalars (lse1, lse2, dkl, kl) from a packed copy: 16 B per query, rows padded to 64 per head -- O(NQ).
  if (B <= 0 || H <= 0 || NQ <= 0) return 0;
  if (!tc_dims(d1, d2)) return 0;   // SIMT path: no workspace
  const long long BH = (long long)B * H;
  if (!bwd_fused_selected(NQ, want_teacher != 0, d1, d2)) return size_t(BH) * size_t(stats_padded_rows(NQ)) * 16;
  // one-visit kernels (mode FUSED, or AUTO with NQ <= 512): + their fp32 dQ accumulators, O(NQ d)
  return stats_bytes_aligned(BH, NQ) + fused_acc_bytes_aligned(BH, NQ, pad_dim(d2)) + (want_teacher ? fused_acc_bytes_aligned(BH, NQ, pad_dim(d1)) : 0);
}

int streamkl_set_fwd_plan(int plan) {
  if (plan < STREAMKL_FWD_AUTO || plan > STREAMKL_FWD_PER_TILE) return STREAMKL_ERR_SHAPE;
  g_fwd_plan = plan;
  return STREAMKL_OK;
}

int streamkl_set_bwd_mode(int mode) {
  if (mode != STREAMKL_BWD_AUTO && mode != STREAMKL_BWD_SEPARATE && mode != STREAMKL_BWD_FUSED) return STREAMKL_ERR_SHAPE;
  g_bwd_mode = mode;
  return STREAMKL_OK;
}

int streamkl_fwd_host(int dtype, const void* Q1, const void* K1, const void* Q2, const void* K2, int B, int H, int NQ, int NK, int d1,
                      int d2, float c1, float c2, int causal, float* kl_rows, float* lse1, float* lse2, streamkl_stream_t stream) {
  return streamkl_fwd_bwd_host(dtype, Q1, K1, Q2, K2, B, H, NQ, NK, d1, d2, c1, c2, causal, nullptr, kl_rows, lse1, lse2, nullptr,
                               nullptr, nullptr, nullptr, stream);
}

int streamkl_fwd_bwd_host(int dtype, const void* Q1, const void* K1, const void* Q2, const void* K2, int B, int H, int NQ, int NK,
                          int d1, int d2, float c1, float c2, int causal, const float* dkl_rows, float* kl_rows, float* lse1,
                          float* lse2, void* dQ1, void* dK1, void* dQ2, void* dK2, streamkl_stream_t stream_) {
  if (dtype != STREAMKL_BF16 && dtype != STREAMKL_F32) return STREAMKL_ERR_DTYPE;
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  Shape s{B, H, NQ, NK, d1, d2, causal ? 1 : 0, c1, c2, (long long)B * (long long)H};
  // host pointers need no 16-byte alignment: validate with aligned stand-ins
  int rc = validate_common(Q1 ? (const void*)16 : nullptr, K1 ? (const void*)16 : nullptr, Q2 ? (const void*)16 : nullptr,
                           K2 ? (const void*)16 : nullptr, s);
  if (rc != STREAMKL_OK) return rc;
  const bool want_bwd = dQ2 != nullptr || dK2 != nullptr;
  if (want_bwd && (!dQ2 || !dK2 || !dkl_rows)) return STREAMKL_ERR_NULLPTR;
  if ((dQ1 == nullptr) != (dK1 == nullptr)) return STREAMKL_ERR_NULLPTR;
  if (!want_bwd && dQ1) return STREAMKL_ERR_NULLPTR;
  if (s.BH == 0 || s.NQ == 0) {
    if (!want_bwd || s.BH == 0) return STREAMKL_OK;
  } else if (!kl_rows || !lse1 || !lse2) {
    return STREAMKL_ERR_NULLPTR;
  }
  if (!device_is_sm100()) return STREAMKL_ERR_CUDA;
  const size_t es = dtype == STREAMKL_BF16 ? 2 : 4;
  const bool teacher = dQ1 != nullptr;
  // per-head sizes: heads are independent, so the batch is cut into groups of whole heads and the upload of group g+1
  // and the download of group g-1 overlap the kernels of group g (three streams, events between them)
  const size_t hq1 = size_t(NQ) * d1 * es, hk1 = size_t(NK) * d1 * es, hq2 = size_t(NQ) * d2 * es, hk2 = size_t(NK) * d2 * es;
  const size_t hrow = size_t(NQ) * sizeof(float);
  const size_t hws = want_bwd ? streamkl_bwd_workspace_bytes(1, 1, NQ, NK, d1, d2, teacher) : 0;
  const long long BH = s.BH;
  long long gs = BH;   // heads per group
  if (BH > 1 && (size_t(d1) * es) % 16 == 0 && (size_t(d2) * es) % 16 == 0 && size_t(BH) * (hq1 + hk1 + hq2 + hk2) >= (64u << 20)) {
    const long long tq = (NQ + kFwdBQ - 1) / kFwdBQ;   // forward CTAs per head
    const long long fill = (2 * 148 + tq - 1) / (tq > 0 ? tq : 1);   // enough CTAs per launch for two waves
    gs = (BH + 7) / 8;
    if (gs < fill) gs = fill;
    if (gs > BH) gs = BH;
  }
  const int G = int((BH + gs - 1) / gs);
  HostStreams& hs = host_streams();
  if (!hs.ok) return STREAMKL_ERR_CUDA;

  AsyncScratch sc(stream);
  uint8_t* bQ1 = static_cast<uint8_t*>(sc.get(BH * hq1));
  uint8_t* bK1 = static_cast<uint8_t*>(sc.get(BH * hk1));
  uint8_t* bQ2 = static_cast<uint8_t*>(sc.get(BH * hq2));
  uint8_t* bK2 = static_cast<uint8_t*>(sc.get(BH * hk2));
  uint8_t* bkl = static_cast<uint8_t*>(sc.get(BH * hrow));
  uint8_t* bl1 = static_cast<uint8_t*>(sc.get(BH * hrow));
  uint8_t* bl2 = static_cast<uint8_t*>(sc.get(BH * hrow));
  uint8_t *bg = nullptr, *gQ1 = nullptr, *gK1 = nullptr, *gQ2 = nullptr, *gK2 = nullptr, *bws = nullptr;
  if (want_bwd) {
    bg = static_cast<uint8_t*>(sc.get(BH * hrow));
    gQ2 = static_cast<uint8_t*>(sc.get(BH * hq2));
    gK2 = static_cast<uint8_t*>(sc.get(BH * hk2));
    bws = static_cast<uint8_t*>(sc.get(BH * hws));
    if (teacher) {
      gQ1 = static_cast<uint8_t*>(sc.get(BH * hq1));
      gK1 = static_cast<uint8_t*>(sc.get(BH * hk1));
    }
  }
  if (!sc.ok) return STREAMKL_ERR_CUDA;
  std::vector<cudaEvent_t> ev(size_t(2 * G + 4), nullptr);
  bool ok = true;
  for (cudaEvent_t& e : ev) ok = ok && cudaEventCreateWithFlags(&e, cudaEventDisableTiming) == cudaSuccess;
  auto cleanup = [&]() { for (cudaEvent_t e : ev) if (e) cudaEventDestroy(e); };
  if (!ok) { cudaGetLastError(); cleanup(); return STREAMKL_ERR_CUDA; }
  cudaEvent_t ev_start = ev[size_t(2 * G)], ev_in_done = ev[size_t(2 * G + 1)], ev_cmp_done = ev[size_t(2 * G + 2)], ev_out_done = ev[size_t(2 * G + 3)];
  // the scratch was allocated in order on `stream`: everything else starts after that point
  ok = ok && cudaEventRecord(ev_start, stream) == cudaSuccess && cudaStreamWaitEvent(hs.in, ev_start, 0) == cudaSuccess &&
       cudaStreamWaitEvent(hs.cmp, ev_start, 0) == cudaSuccess && cudaStreamWaitEvent(hs.out, ev_start, 0) == cudaSuccess;
  auto cp = [&](void* dst, const void* src, size_t n, cudaMemcpyKind kind, cudaStream_t st) {
    return n == 0 || cudaMemcpyAsync(dst, src, n, kind, st) == cudaSuccess;
  };
  const uint8_t *hQ1 = static_cast<const uint8_t*>(Q1), *hK1 = static_cast<const uint8_t*>(K1);
  const uint8_t *hQ2 = static_cast<const uint8_t*>(Q2), *hK2 = static_cast<const uint8_t*>(K2);
  int launches = 0;
  rc = STREAMKL_OK;
  for (int g = 0; g < G && ok && rc == STREAMKL_OK; ++g) {
    const size_t h0 = size_t(g) * size_t(gs);
    const int hn = int(std::min<long long>(gs, BH - (long long)h0));
    // ---- upload (stream `in`)
    ok = ok && cp(bQ1 + h0 * hq1, hQ1 + h0 * hq1, hn * hq1, cudaMemcpyHostToDevice, hs.in) &&
         cp(bK1 + h0 * hk1, hK1 + h0 * hk1, hn * hk1, cudaMemcpyHostToDevice, hs.in) &&
         cp(bQ2 + h0 * hq2, hQ2 + h0 * hq2, hn * hq2, cudaMemcpyHostToDevice, hs.in) &&
         cp(bK2 + h0 * hk2, hK2 + h0 * hk2, hn * hk2, cudaMemcpyHostToDevice, hs.in);
    if (want_bwd) ok = ok && cp(bg + h0 * hrow, reinterpret_cast<const uint8_t*>(dkl_rows) + h0 * hrow, hn * hrow, cudaMemcpyHostToDevice, hs.in);
    ok = ok && cudaEventRecord(ev[size_t(2 * g)], hs.in) == cudaSuccess && cudaStreamWaitEvent(hs.cmp, ev[size_t(2 * g)], 0) == cudaSuccess;
    if (!ok) break;
    // ---- kernels (stream `cmp`): the group is a batch of hn heads
    if (s.NQ > 0) {
      rc = fwd_dispatch(dtype, nullptr, bQ1 + h0 * hq1, bK1 + h0 * hk1, bQ2 + h0 * hq2, bK2 + h0 * hk2, 1, hn, NQ, NK, d1, d2, c1, c2, causal,
                        reinterpret_cast<float*>(bkl + h0 * hrow), reinterpret_cast<float*>(bl1 + h0 * hrow),
                        reinterpret_cast<float*>(bl2 + h0 * hrow), hs.cmp);
      if (rc != STREAMKL_OK) break;
      launches += g_last_launches;
    }
    if (want_bwd) {
      rc = bwd_dispatch(dtype, nullptr, bQ1 + h0 * hq1, bK1 + h0 * hk1, bQ2 + h0 * hq2, bK2 + h0 * hk2, 1, hn, NQ, NK, d1, d2, c1, c2, causal,
                        reinterpret_cast<float*>(bkl + h0 * hrow), reinterpret_cast<float*>(bl1 + h0 * hrow),
                        reinterpret_cast<float*>(bl2 + h0 * hrow), reinterpret_cast<float*>(bg + h0 * hrow),
                        teacher ? gQ1 + h0 * hq1 : nullptr, teacher ? gK1 + h0 * hk1 : nullptr, gQ2 + h0 * hq2, gK2 + h0 * hk2,
                        hws ? bws + h0 * hws : nullptr, hn * hws, hs.cmp);
      if (rc != STREAMKL_OK) break;
      launches += g_last_launches;
    }
    ok = ok && cudaEventRecord(ev[size_t(2 * g + 1)], hs.cmp) == cudaSuccess && cudaStreamWaitEvent(hs.out, ev[size_t(2 * g + 1)], 0) == cudaSuccess;
    // ---- download (stream `out`)
    if (s.NQ > 0)
      ok = ok && cp(reinterpret_cast<uint8_t*>(kl_rows) + h0 * hrow, bkl + h0 * hrow, hn * hrow, cudaMemcpyDeviceToHost, hs.out) &&
           cp(reinterpret_cast<uint8_t*>(lse1) + h0 * hrow, bl1 + h0 * hrow, hn * hrow, cudaMemcpyDeviceToHost, hs.out) &&
           cp(reinterpret_cast<uint8_t*>(lse2) + h0 * hrow, bl2 + h0 * hrow, hn * hrow, cudaMemcpyDeviceToHost, hs.out);
    if (want_bwd) {
      ok = ok && cp(static_cast<uint8_t*>(dQ2) + h0 * hq2, gQ2 + h0 * hq2, hn * hq2, cudaMemcpyDeviceToHost, hs.out) &&
           cp(static_cast<uint8_t*>(dK2) + h0 * hk2, gK2 + h0 * hk2, hn * hk2, cudaMemcpyDeviceToHost, hs.out);
      if (teacher)
        ok = ok && cp(static_cast<uint8_t*>(dQ1) + h0 * hq1, gQ1 + h0 * hq1, hn * hq1, cudaMemcpyDeviceToHost, hs.out) &&
             cp(static_cast<uint8_t*>(dK1) + h0 * hk1, gK1 + h0 * hk1, hn * hk1, cudaMemcpyDeviceToHost, hs.out);
    }
  }
  // join: `stream` continues (and the scratch is returned to the pool) only after all three helper streams are done
  cudaEventRecord(ev_in_done, hs.in); cudaEventRecord(ev_cmp_done, hs.cmp); cudaEventRecord(ev_out_done, hs.out);
  cudaStreamWaitEvent(stream, ev_in_done, 0); cudaStreamWaitEvent(stream, ev_cmp_done, 0); cudaStreamWaitEvent(stream, ev_out_done, 0);
  const bool synced = cudaStreamSynchronize(stream) == cudaSuccess;
  cleanup();
  if (rc != STREAMKL_OK) { cudaGetLastError(); return rc; }
  if (!ok || !synced) { cudaGetLastError(); return STREAMKL_ERR_CUDA; }
  g_last_launches = launches;
  return STREAMKL_OK;
}

int streamkl_host_trim(void) {
  int dev = 0;
  cudaMemPool_t pool;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetDefaultMemPool(&pool, dev) != cudaSuccess ||
      cudaDeviceSynchronize() != cudaSuccess || cudaMemPoolTrimTo(pool, 0) != cudaSuccess) {
    cudaGetLastError();
    return STREAMKL_ERR_CUDA;
  }
  return STREAMKL_OK;
}

int streamkl_last_launch_count(void) { return g_last_launches; }

int streamkl_profile_enable(int on) {
  g_prof_on = on != 0;
  // on > 1: also create that many event pairs now, so that no event is created inside the caller's timed region
  if (on > 1) {
    std::vector<cudaEvent_t> tmp;
    for (int i = 0; i < 2 * on; ++i) { cudaEvent_t e = prof_event(); if (!e) break; tmp.push_back(e); }
    for (cudaEvent_t e : tmp) prof_release(e);
  }
  return STREAMKL_OK;
}

int streamkl_profile_collect(int max_records, int* kernel_ids, float* ms) {
  if (max_records < 0 || (max_records > 0 && (!kernel_ids || !ms))) return STREAMKL_ERR_NULLPTR;
  if (!g_prof) return 0;
  int n = 0, rc = 0;
  for (ProfRecord& r : *g_prof) {
    float t = 0.f;
    if (cudaEventSynchronize(r.b) != cudaSuccess || cudaEventElapsedTime(&t, r.a, r.b) != cudaSuccess) { cudaGetLastError(); rc = STREAMKL_ERR_CUDA; }
    else if (n < max_records) { kernel_ids[n] = r.id; ms[n] = t; ++n; }
    prof_release(r.a);
    prof_release(r.b);
  }
  g_prof->clear();
  return rc < 0 ? rc : n;
}

const char* streamkl_kernel_name(int kernel_id) {
  return (kernel_id >= 0 && kernel_id < KID_COUNT) ? kKernelNames[kernel_id] : "unknown kernel id";
}

const char* streamkl_strerror(int code) {
  switch (code) {
    case STREAMKL_OK: return "ok";
    case STREAMKL_ERR_NULLPTR: return "required pointer is NULL";
    case STREAMKL_ERR_SHAPE: return "unsupported shape (sizes, head dim, or causal with NQ > NK)";
    case STREAMKL_ERR_ALIGN: return "tensor pointer not 16-byte aligned";
    case STREAMKL_ERR_SCALE: return "scale c1/c2 must be finite and > 0";
    case STREAMKL_ERR_WORKSPACE: return "workspace missing or too small";
    case STREAMKL_ERR_CUDA: return "CUDA failure (no sm_100 device, tensor-map, launch, copy or allocation)";
    case STREAMKL_ERR_DTYPE: return "unknown dtype code";
    case STREAMKL_ERR_SCRATCH_LIMIT: return "split-K partials exceed the library's built-in scratch (streamkl_fwd_splitk_noalloc_capacity)";
    default: return "unknown error code";
  }
}

const char* streamkl_version(void) { return "streamkl-b200 0.3 (sm_100a; tcgen05+TMA bf16/fp16, head dims to 256, strided + shared-K-head layouts, persistent / CTA-pair forward plans; SIMT fp32)"; }

}  // extern "C"
