// streamkl_fwd.cu -- launchers of the tcgen05 forward kernel (default grid and split-K + reduce); see streamkl.cu for the C ABI.
#include "streamkl_host.cuh"
#include <algorithm>
#include <atomic>
#include <mutex>
#include <new>

#include "streamkl_fwd_sm100.cuh"
#include "streamkl_fwd_persist_sm100.cuh"

namespace sklh {
namespace {

static_assert(skl::FwdCfg<128, 128>::BQ == kFwdBQ && skl::FwdCfg<64, 64>::BK == kFwdBK, "tile sizes quoted in streamkl_host.cuh");

// splits == 1: the default kernel (grid (bsz, T_Q)).  splits > 1: split-K (grid (bsz, T_Q, W), partial
// statistics to `part`, then the reduce kernel).
// D1 = D2 = 0: the BLOCKED plan with run-time K-block counts (a head dim above 128, padded to 192 / 256).
template <int D1, int D2, bool CAUSAL, bool SPLIT = false, bool MC = false, bool P2 = false>
int launch_fwd_tc(const void* Q1, const void* K1, const void* Q2, const void* K2, const Shape& s, bool f16, float* kl, float* lse1,
                  float* lse2, cudaStream_t stream, int splits = 1, float* part = nullptr) {
  using C = skl::FwdCfg<D1, D2>;
  CUtensorMap tm[4];
  // (cta_group::2 plan: each CTA of a pair loads its own 64 keys of every 128-key block)
  if (!make_maps(tm, Q1, K1, Q2, K2, s, C::BM, P2 ? C::BK / 2 : C::BK, f16)) return STREAMKL_ERR_CUDA;
  const CUtensorMap &tQ1 = tm[0], &tK1 = tm[1], &tQ2 = tm[2], &tK2 = tm[3];
  auto kern = skl::streamkl_fwd_sm100_kernel<D1, D2, CAUSAL, SPLIT, MC, P2>;
  skl::FwdParams p;
  p.kb1 = pad_dim(s.d1) / 64; p.kb2 = pad_dim(s.d2) / 64; p.nring = 0;
  int smem_bytes = 0;
  if constexpr (C::BLOCKED) {
    const int slot = P2 ? C::KBLK / 2 : C::KBLK;
    p.nring = C::ring_blocks(p.kb1, p.kb2, slot);
    if (p.nring < 2) return STREAMKL_ERR_SHAPE;
    smem_bytes = C::smem_bytes(p.kb1, p.kb2, slot);
  } else {
    smem_bytes = C::SMEM_BYTES;
  }
  // (the BLOCKED plan's size depends on the head dims, and the attribute is per function, not per launch: always raise it to the
  // same constant, so that concurrent host threads with different head-dim pairs cannot lower it under one another)
  if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, C::BLOCKED ? C::SMEM_LIMIT : smem_bytes) != cudaSuccess) {
    cudaGetLastError();
    return STREAMKL_ERR_CUDA;
  }
  p.NQ = s.NQ; p.NK = s.NK; p.BH = int(s.BH);
  p.H = s.H; p.G = s.G(); p.fmt16 = f16 ? 0u : 1u; p.act2 = s.act2;
  p.TQ = (s.NQ + C::BQ - 1) / C::BQ;
  p.sc1 = s.c1 * 1.4426950408889634f;
  p.sc2 = s.c2 * 1.4426950408889634f;
  p.kl = kl; p.lse1 = lse1; p.lse2 = lse2;
  const int TK = (s.NK + C::BK - 1) / C::BK;
  p.chunk_steps = SPLIT ? (TK + splits - 1) / splits : TK;       // C_K = ceil(N_K / W), in whole BK-key steps
  p.W = SPLIT ? (TK + p.chunk_steps - 1) / p.chunk_steps : 1;    // no empty trailing chunk
  p.part = part;
  const long long grid = (MC || P2) ? 2LL * ((p.TQ + 1) / 2) * s.BH : (long long)p.TQ * s.BH * p.W;
  if (grid > 0x7fffffffLL) return STREAMKL_ERR_SHAPE;
  {
    ProfScope ps(SPLIT ? KID_FWD_SPLITK_TC : KID_FWD_TC, stream);
    if constexpr (MC || P2) {   // clusters of two CTAs: the Q tiles (2i, 2i+1) of a head share one multicast K stream
      cudaLaunchConfig_t cfg = {};
      cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3(C::THREADS); cfg.dynamicSmemBytes = size_t(smem_bytes); cfg.stream = stream;
      cudaLaunchAttribute at[1];
      at[0].id = cudaLaunchAttributeClusterDimension;
      at[0].val.clusterDim.x = 2; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
      cfg.attrs = at; cfg.numAttrs = 1;
      if (cudaLaunchKernelEx(&cfg, kern, tQ1, tK1, tQ2, tK2, p) != cudaSuccess) { cudaGetLastError(); return STREAMKL_ERR_CUDA; }
    } else {
      kern<<<dim3((unsigned)grid), C::THREADS, smem_bytes, stream>>>(tQ1, tK1, tQ2, tK2, p);
    }
  }
  if (cudaGetLastError() != cudaSuccess) return STREAMKL_ERR_CUDA;
  g_last_launches += 1;
  if (SPLIT) {
    const long long rows = s.BH * (long long)s.NQ;
    {
      ProfScope ps(KID_FWD_SPLITK_REDUCE, stream);
      skl::streamkl_fwd_splitk_reduce_kernel<<<dim3((unsigned)((rows + 127) / 128)), 128, 0, stream>>>(part, s.NQ, p.W, rows, kl, lse1, lse2);
    }
    if (cudaGetLastError() != cudaSuccess) return STREAMKL_ERR_CUDA;
    g_last_launches += 1;
  }
  return STREAMKL_OK;
}

// ---- persistent forward (streamkl_fwd_persist_sm100.cuh): one CTA per SM, dynamic work items
// Scheduler state of the persistent kernel: {next item, finished CTAs} per slot, zero between launches (the last CTA of a launch
// rearms its slot).  Two launches that can be in flight at the same time must not share a slot (they would take each other's
// tickets and skip tiles), so a slot is LEASED: the host records an event behind every launch that used it and hands the slot out
// again only once that event has completed.  When no slot is free (hundreds of launches queued) or the stream is being captured
// into a CUDA graph (a captured launch would keep its slot for as long as the graph lives, and an event recorded during capture
// cannot be queried), the caller runs the per-tile kernel instead: same results bit for bit.
constexpr int kSchedSlots = 1024;
constexpr int kSchedProbe = 16;      // slots examined per launch before giving up
constexpr int kSchedMaxDevices = 64;
__device__ int g_fwd_sched[kSchedSlots][2];

struct SchedLeases {
  std::mutex mu;
  unsigned next = 0;
  cudaEvent_t done[kSchedSlots] = {};   // recorded behind the last launch that used the slot (created on first use)
  bool held[kSchedSlots] = {};          // between acquire() and release(): the launch and its event are being enqueued
};
std::mutex g_sched_mu;
SchedLeases* g_sched_leases[kSchedMaxDevices] = {};

SchedLeases* sched_leases(int dev) {
  if (dev < 0 || dev >= kSchedMaxDevices) return nullptr;
  std::lock_guard<std::mutex> lock(g_sched_mu);
  if (!g_sched_leases[dev]) g_sched_leases[dev] = new (std::nothrow) SchedLeases();
  return g_sched_leases[dev];
}

// a slot no launch in flight is using, or -1
int sched_acquire(SchedLeases& L) {
  std::lock_guard<std::mutex> lock(L.mu);
  for (int probe = 0; probe < kSchedProbe; ++probe) {
    const int i = int(L.next++ % kSchedSlots);
    if (L.held[i]) continue;
    if (!L.done[i]) {
      if (cudaEventCreateWithFlags(&L.done[i], cudaEventDisableTiming) != cudaSuccess) { cudaGetLastError(); L.done[i] = nullptr; return -1; }
    } else if (cudaEventQuery(L.done[i]) != cudaSuccess) {
      cudaGetLastError();   // cudaErrorNotReady: the last launch on this slot has not finished
      continue;
    }
    L.held[i] = true;
    return i;
  }
  return -1;
}

// after the launch (or a failed one): mark the slot busy until everything enqueued on `stream` so far has finished
bool sched_release(SchedLeases& L, int slot, cudaStream_t stream) {
  const bool ok = cudaEventRecord(L.done[slot], stream) == cudaSuccess;
  if (!ok) cudaGetLastError();
  std::lock_guard<std::mutex> lock(L.mu);
  L.held[slot] = false;
  return ok;
}

bool stream_is_capturing(cudaStream_t stream) {
  cudaStreamCaptureStatus st = cudaStreamCaptureStatusNone;
  if (cudaStreamIsCapturing(stream, &st) != cudaSuccess) { cudaGetLastError(); return true; }   // (e.g. the legacy stream during a global capture)
  return st != cudaStreamCaptureStatusNone;
}

// SMs of the current device (asked once per device ordinal; 148 on a B200)
int sm_count() {
  static std::atomic<int> cached[kSchedMaxDevices];
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kSchedMaxDevices) { cudaGetLastError(); return 148; }
  int n = cached[dev].load(std::memory_order_relaxed);
  if (n <= 0) {
    if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) { cudaGetLastError(); return 148; }
    cached[dev].store(n, std::memory_order_relaxed);
  }
  return n;
}

constexpr int kPersistUnavailable = 1;   // launch_fwd_persist: no scheduler slot could be leased -- run the per-tile kernel

template <int D1, int D2, bool CAUSAL>
int launch_fwd_persist(const void* Q1, const void* K1, const void* Q2, const void* K2, const Shape& s, bool f16, float* kl, float* lse1,
                       float* lse2, cudaStream_t stream) {
  using C = skl::FwdPersistCfg<D1, D2>;
  CUtensorMap tm[4];
  if (!make_maps(tm, Q1, K1, Q2, K2, s, C::BM, C::BK, f16)) return STREAMKL_ERR_CUDA;
  auto kern = skl::streamkl_fwd_persist_sm100_kernel<D1, D2, CAUSAL>;
  int dev = 0, sms = 0;
  int* sched = nullptr;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
      cudaGetSymbolAddress(reinterpret_cast<void**>(&sched), g_fwd_sched) != cudaSuccess ||
      cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES) != cudaSuccess) {
    cudaGetLastError();
    return STREAMKL_ERR_CUDA;
  }
  skl::FwdParams p;
  p.kb1 = D1 / 64; p.kb2 = D2 / 64; p.nring = 0;
  p.NQ = s.NQ; p.NK = s.NK; p.BH = int(s.BH);
  p.H = s.H; p.G = s.G(); p.fmt16 = f16 ? 0u : 1u; p.act2 = s.act2;
  p.TQ = (s.NQ + C::BQ - 1) / C::BQ;
  p.sc1 = s.c1 * 1.4426950408889634f;
  p.sc2 = s.c2 * 1.4426950408889634f;
  p.kl = kl; p.lse1 = lse1; p.lse2 = lse2;
  p.W = 1; p.chunk_steps = 0; p.part = nullptr;
  const long long total = (long long)p.TQ * s.BH;
  if (total > 0x7fffffffLL) return STREAMKL_ERR_SHAPE;
  const int grid = int(total < sms ? total : sms);
  SchedLeases* leases = sched_leases(dev);
  const int slot = leases ? sched_acquire(*leases) : -1;
  if (slot < 0) return kPersistUnavailable;
  sched += 2 * slot;
  {
    ProfScope ps(KID_FWD_TC, stream);
    kern<<<dim3((unsigned)grid), C::THREADS, C::SMEM_BYTES, stream>>>(tm[0], tm[1], tm[2], tm[3], p, sched);
  }
  const bool launched = cudaGetLastError() == cudaSuccess;
  if (!sched_release(*leases, slot, stream) || !launched) return STREAMKL_ERR_CUDA;
  g_last_launches += 1;
  return STREAMKL_OK;
}

}  // namespace

int fwd_tc_launch(const void* Q1, const void* K1, const void* Q2, const void* K2, const Shape& s, bool f16, float* kl, float* lse1, float* lse2,
                  cudaStream_t stream, int splits, float* part) {
  int p1 = pad_dim(s.d1), p2 = pad_dim(s.d2);
  if (p1 > 128 || p2 > 128) p1 = p2 = 0;   // a wide head dim: the BLOCKED plan (run-time K-block counts)
  // the persistent plan: fixed plans (head dims <= 128), default grid
  // Measured rule of the default plan (profiles/r02h_persistent.md): the persistent kernel wins where tiles are short -- its gain is
  // the time between tiles -- and there are enough of them to keep every SM busy for several items: at most 64 steps per tile on
  // average (N_K <= 16K causal, 8K otherwise) and at least two items per SM.  Long tiles (cfg 4) run 1 % faster one CTA per tile.
  const int TQ = (s.NQ + kFwdBQ - 1) / kFwdBQ, TK = (s.NK + kFwdBK - 1) / kFwdBK;
  const long long tiles = (long long)s.BH * TQ;
  // key steps per Q tile, averaged over the head's tiles.  Causal tile t (rows q0 = t*BQ ...) streams the keys up to its last row's
  // frontier q0 + BQ - 1 + (NK - NQ): ceil of that over BK steps, at most TK -- an arithmetic series in t until it saturates at TK
  // (NQ << NK: every tile streams at least NK - NQ keys, so the average is close to TK, not TK / 2)
  long long sum_steps = (long long)TQ * TK;
  if (s.causal) {
    sum_steps = 0;
    for (int t = 0; t < TQ; ++t) sum_steps += std::min<long long>(TK, ((long long)t * kFwdBQ + kFwdBQ - 1 + (s.NK - s.NQ)) / kFwdBK + 1);
  }
  const long long avg_steps = TQ > 0 ? sum_steps / TQ : 0;   // (rounded down: NQ = NK = 16K causal is 64.5 -> 64, inside the rule)
  bool persist_auto = g_fwd_plan == STREAMKL_FWD_AUTO && avg_steps <= 64 && p1 != 0 && splits <= 1;
  if (persist_auto) persist_auto = tiles >= 2LL * sm_count();   // at least two items per SM of the device that will run it
  if ((g_fwd_plan == STREAMKL_FWD_PERSISTENT || persist_auto) && splits <= 1 && p1 != 0 && !stream_is_capturing(stream)) {
    int rc = kPersistUnavailable;
#define SKL_FWD_P_CASE(A, Bd)                                                                                             \
    if (p1 == A && p2 == Bd)                                                                                              \
      rc = s.causal ? launch_fwd_persist<A, Bd, true>(Q1, K1, Q2, K2, s, f16, kl, lse1, lse2, stream)                      \
                    : launch_fwd_persist<A, Bd, false>(Q1, K1, Q2, K2, s, f16, kl, lse1, lse2, stream);
    SKL_FWD_P_CASE(128, 128)
    SKL_FWD_P_CASE(128, 64)
    SKL_FWD_P_CASE(64, 128)
    SKL_FWD_P_CASE(64, 64)
#undef SKL_FWD_P_CASE
    if (rc != kPersistUnavailable) return rc;   // (no free scheduler slot: the per-tile kernel below, bit-identical)
  }
  // the multicast pair plan (streamkl_set_fwd_plan): the default grid only, and only when a head has a second Q tile to pair
  const bool mc = g_fwd_plan == STREAMKL_FWD_MULTICAST && splits <= 1 && s.NQ > skl::FwdCfg<64, 64>::BQ;
  // the cta_group::2 plan: wide head dims only (BLOCKED plan), default grid
  if (g_fwd_plan == STREAMKL_FWD_PAIR_MMA && splits <= 1 && p1 == 0 && s.NQ > skl::FwdCfg<64, 64>::BQ)
    return s.causal ? launch_fwd_tc<0, 0, true, false, false, true>(Q1, K1, Q2, K2, s, f16, kl, lse1, lse2, stream)
                    : launch_fwd_tc<0, 0, false, false, false, true>(Q1, K1, Q2, K2, s, f16, kl, lse1, lse2, stream);
#define SKL_FWD_MC_CASE(A, Bd)                                                                                                    \
  if (mc && p1 == A && p2 == Bd)                                                                                                  \
    return s.causal ? launch_fwd_tc<A, Bd, true, false, true>(Q1, K1, Q2, K2, s, f16, kl, lse1, lse2, stream)                     \
                    : launch_fwd_tc<A, Bd, false, false, true>(Q1, K1, Q2, K2, s, f16, kl, lse1, lse2, stream);
  SKL_FWD_MC_CASE(128, 128)
  SKL_FWD_MC_CASE(128, 64)
  SKL_FWD_MC_CASE(64, 128)
  SKL_FWD_MC_CASE(64, 64)
  SKL_FWD_MC_CASE(0, 0)
#undef SKL_FWD_MC_CASE
#define SKL_FWD_CASE(A, Bd)                                                                                                       \
  if (p1 == A && p2 == Bd) {                                                                                                      \
    if (splits > 1)                                                                                                               \
      return s.causal ? launch_fwd_tc<A, Bd, true, true>(Q1, K1, Q2, K2, s, f16, kl, lse1, lse2, stream, splits, part)            \
                      : launch_fwd_tc<A, Bd, false, true>(Q1, K1, Q2, K2, s, f16, kl, lse1, lse2, stream, splits, part);          \
    return s.causal ? launch_fwd_tc<A, Bd, true>(Q1, K1, Q2, K2, s, f16, kl, lse1, lse2, stream)                                  \
                    : launch_fwd_tc<A, Bd, false>(Q1, K1, Q2, K2, s, f16, kl, lse1, lse2, stream);                                \
  }
  SKL_FWD_CASE(128, 128)
  SKL_FWD_CASE(128, 64)
  SKL_FWD_CASE(64, 128)
  SKL_FWD_CASE(64, 64)
  SKL_FWD_CASE(0, 0)
#undef SKL_FWD_CASE
  return STREAMKL_ERR_SHAPE;
}

}  // namespace sklh
