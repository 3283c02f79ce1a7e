// streamkl_host.cuh -- host-side declarations shared by the translation units of libstreamkl.so (one per kernel family, so that
// they compile in parallel): problem description, tensor-map construction, per-launch profiling scope, and the launch
// dispatchers each family exports to the C-ABI glue in streamkl.cu.  Nothing here is part of the public interface.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>

#include <cstddef>
#include <cstdint>

#include "../../include/streamkl.h"

namespace sklh {

extern thread_local int g_fwd_plan;        // streamkl_set_fwd_plan: STREAMKL_FWD_SINGLE | STREAMKL_FWD_MULTICAST
extern thread_local int g_last_launches;   // kernels launched by the current streamkl_* call (streamkl_last_launch_count)

// ---- optional per-kernel timing (streamkl_profile_*): CUDA events recorded on the launch stream around every kernel
enum KernelId { KID_FWD_TC = 0, KID_BWD_DQ_TC, KID_BWD_DK_TC, KID_FWD_SIMT, KID_BWD_DQ_SIMT, KID_BWD_DK_SIMT, KID_BWD_STATS, KID_FWD_SPLITK_TC, KID_FWD_SPLITK_REDUCE, KID_BWD_FUSED_TC, KID_BWD_DQ_CONVERT, KID_BWD_DQ_WIDE, KID_BWD_DK_WIDE, KID_COUNT };
struct ProfScope {  // brackets ONE kernel launch; a no-op unless profiling is enabled on this thread (defined in streamkl.cu)
  cudaStream_t st;
  cudaEvent_t b = nullptr;
  ProfScope(int id, cudaStream_t s);
  ~ProfScope();
};

// Element strides {batch, head, row} of one tensor (the head dimension is contiguous).
struct Strides { long long b, h, n; };

struct Shape {
  int B, H, NQ, NK, d1, d2, causal;
  float c1, c2;
  long long BH;
  // layout (streamkl_layout): K heads, element strides of Q1, K1, Q2, K2 (gradients share their input's strides)
  int HK = 0;
  int act2 = 0;   // student activation (streamkl_layout::student_activation)
  Strides q1{}, k1{}, q2{}, k2{};
  bool default_layout = true;
  int G() const { return HK > 0 ? H / HK : 1; }
};

// tile sizes of the forward kernel (the same for every head-dim pair; static_assert'ed against FwdCfg in streamkl_fwd.cu)
constexpr int kFwdBQ = 128, kFwdBK = 128;
// queries per head in the padded per-query scalar array of the backward (= skl::bwd_stats_padded_rows)
constexpr long long stats_padded_rows(long long NQ) { return (NQ + 63) / 64 * 64; }
// the tensor-core kernels work on head dims that are multiples of 64 (fixed plans: 64 and 128; run-time K-block counts above
// that: 192 and 256); anything else runs zero-padded to the next multiple
inline int pad_dim(int d) { return d <= 64 ? 64 : (d + 63) / 64 * 64; }
constexpr int kMaxTcDim = 256;
inline bool wide_dims(int d1, int d2) { return pad_dim(d1) > 128 || pad_dim(d2) > 128; }

// 4-D maps {d, N, heads, B} of the four inputs, box = {64 elements, rows, 1, 1}, 128-byte swizzle, zero OOB fill
bool make_maps(CUtensorMap (&t)[4], const void* Q1, const void* K1, const void* Q2, const void* K2, const Shape& s, int rows_q, int rows_k,
               bool f16);

// ---- launch dispatchers of the tensor-core kernel families (each in its own translation unit)
// forward: splits == 1 the default kernel, > 1 split-K + reduce (streamkl_fwd.cu)
int fwd_tc_launch(const void* Q1, const void* K1, const void* Q2, const void* K2, const Shape& s, bool f16, float* kl, float* lse1, float* lse2,
                  cudaStream_t stream, int splits, float* part);
// backward pre-pass B1 (packed per-query scalars) and the two owner kernels (streamkl_bwd_q.cu / streamkl_bwd_k.cu)
int bwd_stats_launch(const Shape& s, const float* kl, const float* lse1, const float* lse2, const float* dkl, void* stats, cudaStream_t stream);
int bwd_tc_owner_q_launch(const void* Q1, const void* K1, const void* Q2, const void* K2, const Shape& s, bool f16, const void* stats, void* dQ1,
                          void* dQ2, cudaStream_t stream);
int bwd_tc_owner_k_launch(const void* Q1, const void* K1, const void* Q2, const void* K2, const Shape& s, bool f16, const void* stats, void* dK1,
                          void* dK2, cudaStream_t stream);
// the owner kernels for head dims above 128 (streamkl_bwd_wide_q.cu / streamkl_bwd_wide_k.cu): one or two passes per owner side
int bwd_wide_owner_q_launch(const void* Q1, const void* K1, const void* Q2, const void* K2, const Shape& s, bool f16, const void* stats, void* dQ1,
                            void* dQ2, cudaStream_t stream);
int bwd_wide_owner_k_launch(const void* Q1, const void* K1, const void* Q2, const void* K2, const Shape& s, bool f16, const void* stats, void* dK1,
                            void* dK2, cudaStream_t stream);
// one one-visit pass (student: dS2 -> dQ2, dK2; teacher: dS1 -> dQ1, dK1) + its dQ convert (streamkl_bwd_fused.cu)
int bwd_tc_fused_launch(const void* Q1, const void* K1, const void* Q2, const void* K2, const Shape& s, bool f16, bool teacher_pass,
                        const void* stats, float* dq_acc, void* dQ, void* dK, cudaStream_t stream);

}  // namespace sklh
