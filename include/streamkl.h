/*
 * streamkl.h -- C ABI of the B200-native StreamKL hot path (arxiv/paper_2606_20005).
 *
 * The operation.  For every (batch b, head h) and query row i, with logits
 *     s_t[j] = c_t * <Q_t[b,h,i,:], K_t[b,h,j,:]>,   t in {1,2}          (sqrt(d) scale = c_t)
 * over the visible keys V_i (all keys, or causal j <= i + (NK-NQ)), the library computes
 *     lse_t[i] = log sum_{j in V_i} exp(s_t[j])                             (Eq.4)
 *     kl[i]    = KL(P1 || P2) = sum_j P1[j] (log P1[j] - log P2[j])         (Eq.1)
 * in ONE streaming pass over key tiles via  kl = acc/l1 + lse2 - lse1,  acc = sum_j e^{s1-m1}(s1-s2)
 * (Eq.8; Algorithm 1; rescaling invariant Eq.9-10),
 * and, in the backward pass, by tile-wise recomputation from the saved lse:
 *     dS2 = g (P2 - P1)                      -> dQ2 = c2 dS2 K2,  dK2 = c2 dS2^T Q2   (Eq.2 :64; Alg.2 :224-234; :294)
 *     dS1 = g P1 ((s1-s2) - (lse1-lse2) - kl) -> dQ1 = c1 dS1 K1,  dK1 = c1 dS1^T Q1   (Eq.3 :69; Eq.12 :304; Alg.3 :255-286; :309)
 * with g = dkl_rows[i] the upstream gradient (dL in Alg.2/3).  No N_Q x N_K intermediate is ever written to HBM.
 *
 * Conventions (all entry points):
 *  - Tensors are contiguous row-major [B][H][N][d] ("bsz" = B*H flattened) unless a streamkl_layout says
 *    otherwise (strided tensors, K heads shared by groups of query heads: the `*_ex` entry points); per-row vectors are
 *    always contiguous [B][H][NQ] float32.  Outputs are in natural-log units.
 *  - The plain entry points take bf16, `*_f32` fp32, `*_ex` the element type named in the layout (bf16 / fp16 / fp32); gradients
 *    come back in the input type (one rounding from fp32 accumulators).  All accumulation is fp32.  16-bit inputs with d1, d2
 *    multiples of 8 up to 256 run the tcgen05/TMA kernels (head dims zero-padded to the next multiple of 64 inside the kernels;
 *    above 128 the forward streams K in 64-element K-blocks and the backward differentiates one distribution per launch when
 *    d1 + d2 > 256 padded); every other case (fp32 inputs, head dims up to 256 that are not multiples of 8) runs the SIMT fp32 kernels.
 *  - Device entry points take DEVICE pointers owned by the caller; the library never allocates, frees or
 *    retains them, and only enqueues work on `stream` (asynchronous; device faults surface at the caller's next
 *    synchronisation).  `*_host` entry points take HOST pointers, allocate their own device scratch, copy in,
 *    run, copy back and synchronise before returning.
 *  - Return value: 0 (STREAMKL_OK) or a negative STREAMKL_ERR_* code.  Argument errors (every code but
 *    STREAMKL_ERR_CUDA) are detected before anything is enqueued: such a call enqueues nothing and writes nothing.  A
 *    STREAMKL_ERR_CUDA (tensor-map encode, launch or copy failure) can surface after earlier kernels of the same call were
 *    enqueued; the outputs are then unspecified.  The library never throws, prints or exits.  There is no CPU fallback: on a machine without
 *    an sm_100 GPU every compute entry point returns STREAMKL_ERR_CUDA.
 *  - Thread-safe for concurrent calls on distinct streams.
 *  - Shapes: B,H >= 0 (B*H == 0 or NQ == 0 is a successful no-op), NK >= 1, 1 <= d1,d2 <= 256,
 *    causal requires NQ <= NK (bottom-right aligned mask; rows would otherwise have empty support).
 *    c1,c2 must be finite and > 0.  Pointers must be 16-byte aligned (TMA).
 */
#ifndef STREAMKL_H_
#define STREAMKL_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

/* A CUDA stream handle (cudaStream_t / CUstream) passed as an opaque pointer; NULL = the legacy default stream. */
typedef void* streamkl_stream_t;

enum {
  STREAMKL_OK = 0,
  STREAMKL_ERR_NULLPTR = -1,   /* a required pointer is NULL */
  STREAMKL_ERR_SHAPE = -2,     /* negative size, NK < 1, d out of range, causal with NQ > NK, B*H*N overflow */
  STREAMKL_ERR_ALIGN = -3,     /* a tensor pointer is not 16-byte aligned */
  STREAMKL_ERR_SCALE = -4,     /* c1 or c2 is not finite and > 0 */
  STREAMKL_ERR_WORKSPACE = -5, /* workspace NULL or smaller than streamkl_bwd_workspace_bytes() */
  STREAMKL_ERR_CUDA = -6,      /* no sm_100 device, tensor-map encode / launch / copy / allocation failure */
  STREAMKL_ERR_DTYPE = -7,     /* unknown dtype code */
  STREAMKL_ERR_SCRATCH_LIMIT = -8 /* streamkl_fwd_splitk_noalloc: the partials of this shape and split count exceed the built-in scratch */
};

enum { STREAMKL_BF16 = 0, STREAMKL_F32 = 1, STREAMKL_F16 = 2 };

/*
 * Forward (Algorithm 1).  Device pointers.
 *   Q1 [B][H][NQ][d1], K1 [B][H][NK][d1], Q2 [B][H][NQ][d2], K2 [B][H][NK][d2]  -- read only, `dtype` elements
 *   kl_rows, lse1, lse2 [B][H][NQ] float32 -- overwritten (the 3*NQ scalars of PAPER.md:216-218)
 * Extra HBM: none (O(NQ) outputs only).
 */
int streamkl_fwd(const void* Q1, const void* K1, const void* Q2, const void* K2,
                 int B, int H, int NQ, int NK, int d1, int d2, float c1, float c2, int causal,
                 float* kl_rows, float* lse1, float* lse2, streamkl_stream_t stream);          /* bf16 inputs */
int streamkl_fwd_f32(const void* Q1, const void* K1, const void* Q2, const void* K2,
                     int B, int H, int NQ, int NK, int d1, int d2, float c1, float c2, int causal,
                     float* kl_rows, float* lse1, float* lse2, streamkl_stream_t stream);      /* fp32 inputs */

/*
 * Layouts beyond contiguous [B][H][N][d] (the paper itself only has [bsz, N, d]).
 *   dtype      : STREAMKL_BF16 | STREAMKL_F16 (| STREAMKL_F32: default layout only) -- element type of Q1,K1,Q2,K2 and of the gradients.
 *   kv_heads   : HK, the number of K heads; 0 = H.  H must be a multiple of HK; query head h reads K head h / (H/HK) ("grouped-query"
 *                sharing; K tensors are then [B][HK][NK][d] and dK sums over the H/HK query heads of each group).
 *   *_stride   : ELEMENT strides {batch, head, row} of each input; the head dimension is contiguous (stride 1).  All zero = the
 *                contiguous default for that tensor ([B][H][N][d], or [B][HK][NK][d] for K).  E.g. a [B][N][H][d] tensor is
 *                {N*H*d, d, H*d}.  Strides must be multiples of 8 elements (16 bytes, TMA) and the row stride >= d.
 *                dQ_t is written with Q_t's strides, dK_t with K_t's; kl_rows / lse / dkl_rows stay contiguous [B][H][NQ].
 *                The forward also accepts batch / head stride 0 (a broadcast tensor).  The backward does not: a tensor that receives a
 *                gradient (Q2, K2; Q1, K1 with teacher gradients) must address disjoint rows for distinct (b, h, n) -- no zero or
 *                self-overlapping strides -- because its gradient is stored, not summed, through the same strides
 *                (STREAMKL_ERR_SHAPE otherwise; to share K across query heads use kv_heads, which does sum).
 *   student_activation : SURVEY 8(f) NEXT-4, "Generalizability beyond Softmax" ("the ReLU variant used in the indexer
 *                training of DeepSeek-V3.2"; the paper prints no formula, so this is the library's reading, R23).
 *                STREAMKL_ACT_RELU: the student's logit is s2[j] = relu(c2 <Q2[i], K2[j]>) -- that indexer's score with one head and
 *                unit weight -- and P2 = softmax_j(s2) as before; kl / lse2 are those of this P2, and the student's logit gradient
 *                is gated by relu': dS2 = g (P2 - P1) 1[<Q2[i],K2[j]> > 0].  The teacher side (P1, dS1 of Eq.3) is unchanged.
 * Non-default strides, kv_heads and activations need the tensor-core path: 16-bit dtype and d1, d2 multiples of 8 up to 256 (STREAMKL_ERR_SHAPE
 * otherwise).  Head dims that are not multiples of 64 run zero-padded to the next multiple inside the kernels (TMA zero fill): the
 * results are exact, the padded columns cost tensor work.
 */
enum { STREAMKL_ACT_NONE = 0, STREAMKL_ACT_RELU = 1 };
typedef struct streamkl_layout {
  int dtype;
  int kv_heads;
  long long q1_stride[3], k1_stride[3], q2_stride[3], k2_stride[3];
  int student_activation;   /* STREAMKL_ACT_NONE | STREAMKL_ACT_RELU, see below */
} streamkl_layout;

/* streamkl_fwd / streamkl_bwd with an explicit layout (NULL = bf16, contiguous, HK = H: identical to the plain entry points). */
int streamkl_fwd_ex(const streamkl_layout* layout, const void* Q1, const void* K1, const void* Q2, const void* K2,
                    int B, int H, int NQ, int NK, int d1, int d2, float c1, float c2, int causal,
                    float* kl_rows, float* lse1, float* lse2, streamkl_stream_t stream);
int streamkl_bwd_ex(const streamkl_layout* layout, const void* Q1, const void* K1, const void* Q2, const void* K2,
                    int B, int H, int NQ, int NK, int d1, int d2, float c1, float c2, int causal,
                    const float* kl_rows, const float* lse1, const float* lse2, const float* dkl_rows,
                    void* dQ1, void* dK1, void* dQ2, void* dK2,
                    void* workspace, size_t workspace_bytes, streamkl_stream_t stream);

/*
 * Split-K forward for small NQ (Eq.11; bf16 -- other layouts: streamkl_fwd_splitk_ex below -- d1,d2 multiples of 8 up to 256).  The key range is cut into W
 * contiguous chunks of C_K = 128*ceil(ceil(NK/128)/W) keys (the paper's ceil(NK/W), rounded up to whole 128-key tiles);
 * the grid becomes (bsz, T_Q, W); every CTA writes its chunk's partial statistics (m1,l1,m2,l2,acc) -- 5 floats per
 * row and chunk -- to `workspace`, and a reduce kernel merges them with Eq.11 ((m2,l2) merged the same way) and
 * finishes Alg.1 lines 13-15.  Same outputs as streamkl_fwd up to fp32 summation order.
 *   splits    : W; <= 0 selects it adaptively (streamkl_fwd_splitk_splits with the default target); clamped to
 *               ceil(NK/128); W = 1 launches the default kernel and touches no workspace.
 *   workspace : device scratch of at least streamkl_fwd_splitk_workspace_bytes(B,H,NQ,W) bytes, 16-byte aligned.
 * Other head dims run the unsplit SIMT kernel.  Error behaviour as streamkl_fwd, plus STREAMKL_ERR_WORKSPACE.
 */
int streamkl_fwd_splitk(const void* Q1, const void* K1, const void* Q2, const void* K2,
                        int B, int H, int NQ, int NK, int d1, int d2, float c1, float c2, int causal, int splits,
                        float* kl_rows, float* lse1, float* lse2,
                        void* workspace, size_t workspace_bytes, streamkl_stream_t stream);
/* Split-K with an explicit layout (NULL = streamkl_fwd_splitk): fp16, strided tensors (e.g. a [B][N][H][d] key cache), K heads shared by
 * groups of query heads (kv_heads: decode against a grouped KV cache -- the H/HK query heads of a group stream the same K head, which
 * HBM serves once and the L2 serves to the rest while their CTAs run together) and the ReLU student.  Partials and outputs are laid
 * out by QUERY head as before ([B][H]...), so the workspace size does not depend on kv_heads.  fp32 runs the unsplit SIMT kernel
 * (default layout only). */
int streamkl_fwd_splitk_ex(const streamkl_layout* layout, const void* Q1, const void* K1, const void* Q2, const void* K2,
                           int B, int H, int NQ, int NK, int d1, int d2, float c1, float c2, int causal, int splits,
                           float* kl_rows, float* lse1, float* lse2,
                           void* workspace, size_t workspace_bytes, streamkl_stream_t stream);
/* Adaptive split selection, pure host arithmetic: P_base = B*H*ceil(NQ/128) CTAs of the default kernel;
 * returns 1 if P_base >= p_target, else min(floor(p_target/P_base), ceil(NK/128)).  p_target <= 0 means 148 = one CTA
 * per SM of a B200, i.e. one full wave (the paper's "typically 128 or 256" was for 108/132-SM parts). */
int streamkl_fwd_splitk_splits(int B, int H, int NQ, int NK, int p_target);
/* B*H*splits*5*NQ floats; 0 when splits <= 1. */
size_t streamkl_fwd_splitk_workspace_bytes(int B, int H, int NQ, int splits);

/*
 * Split-K forward for callers that cannot allocate device memory: the same two kernels as streamkl_fwd_splitk (PAPER.md:236-249,
 * Eq.11), same arguments minus the workspace, same results bit for bit for the same W.
 *
 * Who this is for.  streamkl_fwd_splitk needs a caller-owned device buffer for the per-chunk partial statistics.  Some callers
 * have no way to get one at the point of the call: an operator plugged into a serving engine or inference runtime that hands its
 * plugins a fixed arena and forbids driver allocations inside the execute callback; a decode loop with a latency budget, where
 * cudaMalloc / cudaFree would stall every stream of the device; a process whose share of HBM was fixed at start-up (a memory
 * cap per client, or a co-tenant that has already claimed the rest), where a late allocation simply fails.  Small N_Q against a
 * long key cache -- decode -- is exactly where split-K is used, so this is the one entry point that gets such a variant.
 *
 * How.  The partials go to a fixed array of STREAMKL_NOALLOC_SCRATCH_BYTES (4 MiB) that is part of the library's device image:
 * every GPU on which this process uses the library holds those 4 MiB from module load until the process exits, whether or not
 * this function is ever called.  The call itself performs no cudaMalloc, cudaFree, cudaMallocAsync or other allocating call
 * (per-kernel profiling, streamkl_profile_enable, creates events: leave it off -- its default -- on such a path).
 *   splits : W as in streamkl_fwd_splitk.  The limit is  B*H*W*5*NQ*4 bytes <= STREAMKL_NOALLOC_SCRATCH_BYTES  (= the value of
 *            streamkl_fwd_splitk_workspace_bytes; e.g. B*H = 32 heads, NQ = 128, W up to 51; or NQ = 1, B*H = 1024, W up to
 *            204).  An explicit W beyond the limit returns STREAMKL_ERR_SCRATCH_LIMIT and enqueues nothing -- the array is
 *            never grown or replaced.  splits <= 0 (adaptive) picks the paper's W and lowers it until it fits; W = 1 and head
 *            dims off the tensor-core path run the unsplit kernels, which use no scratch at all.
 * First call on each device: the library asks the runtime for the array's address on the device that is current (a symbol lookup,
 * no allocation; it also makes the runtime load the library's device code if this is the first use) and remembers it per device
 * ordinal (up to 64).  Make that first call during set-up, outside any stream capture, with the device you will run on current;
 * later calls on that device do no lookup.
 * Sharing.  Every call on a device, from every stream and host thread, uses the SAME array, and the array keeps whatever the last
 * call wrote.  Nothing needs clearing between calls -- each call overwrites every slot it later reads -- but two calls whose
 * kernels can run at the same time on one GPU (different streams without an ordering between them) overwrite each other's
 * partials and both results are garbage, silently.  Order such calls on one stream or with events; callers that need
 * concurrent split-K calls must use streamkl_fwd_splitk with one workspace per call in flight.
 * Other errors as streamkl_fwd_splitk.  bf16, contiguous [B][H][N][d] only, like streamkl_fwd_splitk.
 */
#define STREAMKL_NOALLOC_SCRATCH_BYTES (4u << 20)
int streamkl_fwd_splitk_noalloc(const void* Q1, const void* K1, const void* Q2, const void* K2,
                                int B, int H, int NQ, int NK, int d1, int d2, float c1, float c2, int causal, int splits,
                                float* kl_rows, float* lse1, float* lse2, streamkl_stream_t stream);
/* STREAMKL_NOALLOC_SCRATCH_BYTES of the library that is actually loaded (for callers that bind at run time). */
size_t streamkl_fwd_splitk_noalloc_capacity(void);

/*
 * Backward (Algorithms 2/3 and their K-tile-owner transposes).
 *   kl_rows, lse1, lse2 : the forward's outputs;  dkl_rows [B][H][NQ] float32 upstream gradient (required).
 *   dQ2 [B][H][NQ][d2], dK2 [B][H][NK][d2] : required, OVERWRITTEN (not accumulated), input dtype.
 *   dQ1 [B][H][NQ][d1], dK1 [B][H][NK][d1] : both NULL => teacher frozen (Setting 1 only); both non-NULL =>
 *                                            Setting 2 gradients too.  Exactly one NULL is STREAMKL_ERR_NULLPTR.
 *   workspace : device scratch of at least streamkl_bwd_workspace_bytes(...) bytes (may be NULL when that is 0).
 * dK is always accumulated atomic-free by K-tile ownership.  dQ: by Q-tile ownership (deterministic, no atomics) under
 * STREAMKL_BWD_SEPARATE; by fp32 atomics under the one-visit strategy, which the default mode selects for small NQ (below).
 */
int streamkl_bwd(const void* Q1, const void* K1, const void* Q2, const void* K2,
                 int B, int H, int NQ, int NK, int d1, int d2, float c1, float c2, int causal,
                 const float* kl_rows, const float* lse1, const float* lse2, const float* dkl_rows,
                 void* dQ1, void* dK1, void* dQ2, void* dK2,
                 void* workspace, size_t workspace_bytes, streamkl_stream_t stream);           /* bf16 */
int streamkl_bwd_f32(const void* Q1, const void* K1, const void* Q2, const void* K2,
                     int B, int H, int NQ, int NK, int d1, int d2, float c1, float c2, int causal,
                     const float* kl_rows, const float* lse1, const float* lse2, const float* dkl_rows,
                     void* dQ1, void* dK1, void* dQ2, void* dK2,
                     void* workspace, size_t workspace_bytes, streamkl_stream_t stream);       /* fp32 */

/*
 * Backward strategy, per calling thread.  The tcgen05 path has two:
 *   STREAMKL_BWD_SEPARATE : a Q-owner kernel (dQ) and a K-owner kernel (dK); every output tile has one owner, no atomics,
 *                           bit-reproducible.
 *   STREAMKL_BWD_FUSED    : one-visit K-owner kernels: a pass visits every tile pair once, keeps dK in place and adds its dQ
 *                           contributions with fp32 atomics into the workspace, then one rounding to the output dtype.  One
 *                           pass for the student (dQ2, dK2: all of Setting 1 -- half the logit recomputation and exps of the
 *                           separate kernels), a second one for the teacher when dQ1, dK1 are requested.  dQ is reproducible
 *                           only up to fp32 summation order.
 *   STREAMKL_BWD_AUTO     : (default) FUSED where it was measured faster on B200, else SEPARATE: (a) small NQ -- NQ <= 512 without
 *                           teacher gradients, NQ <= 256 with them (the paper's rule T_Q*C <= T_K, with the crossover
 *                           found independent of T_K); (b) a frozen teacher with a narrow student at long context -- no teacher
 *                           gradients, d2 <= 64, NQ >= 32768: 7-11 % faster (profiles/r03_bwd_strategies_large.md), at the price of
 *                           the fp32 dQ2 accumulator (4*NQ*64 bytes per head) in the workspace.  NOTE: AUTO is therefore NOT
 *                           bit-reproducible in cases (a) and (b); select STREAMKL_BWD_SEPARATE where that matters.
 * Head dims above 128 always run the owner kernels (deterministic) whatever the mode: one launch per owner side when the
 * gradient accumulators of everything requested fit TMEM together (d1 + d2 <= 256 after padding to multiples of 64, or no
 * teacher gradients), else a student launch and a teacher launch per owner side.
 * Returns STREAMKL_OK, or STREAMKL_ERR_SHAPE for an unknown mode.
 */
enum { STREAMKL_BWD_AUTO = 0, STREAMKL_BWD_SEPARATE = 1, STREAMKL_BWD_FUSED = 2 };
int streamkl_set_bwd_mode(int mode);

/*
 * Forward plan of the default (unsplit) tcgen05 kernel, per calling thread (SURVEY 7.1 step 5 "persistent scheduling", 8(f) NEXT-3
 * "2-CTA / multicast variants").  Every plan computes each row with the same arithmetic in the same order: results are bit-identical.
 *   STREAMKL_FWD_AUTO       : (default) PER_TILE, or PERSISTENT where the measured rule says it wins: head dims <= 128, at most 64 key
 *                             steps per Q tile on average (N_K <= 16K causal, <= 8K unmasked) and at least two Q tiles per SM.
 *   STREAMKL_FWD_PER_TILE   : one CTA per 128-row Q tile (grid bsz x T_Q), each streaming the head's K tiles on its own.
 *   STREAMKL_FWD_PERSISTENT : one CTA per SM loops over the Q tiles (same order, taken from an atomic counter): TMEM and barriers are
 *                             set up once, the next tile's Q / K loads and first MMAs run under the previous tile's last softmax steps.
 *                             Measured on B200: cfg 3 (16K) forward -6..9 %, cfg 2 (4K) -8 %, cfg 4 (64K) +1..2 % (slower).  Head dims
 *                             above 128 run PER_TILE.
 *   STREAMKL_FWD_MULTICAST  : clusters of two CTAs own the Q tiles (2i, 2i+1) of a head and share ONE K stream -- each CTA's
 *                             producer loads half of every stage's K-blocks with TMA multicast into both rings, a stage is
 *                             refilled once both CTAs' MMAs on it have retired.  Half the L2 -> SM traffic.  Measured a tie for head
 *                             dims <= 128 and 6-8 % slower above (the pair runs in lock step on a shallow ring): never chosen by AUTO.
 *   STREAMKL_FWD_PAIR_MMA   : head dims above 128 only (PER_TILE otherwise): the pair issues ONE tcgen05.mma.cta_group::2 per K-slice --
 *                             M = 256 (each CTA's 128 query rows, logits into each CTA's own TMEM), each CTA holding 64 of the 128 keys of
 *                             a K-block, so the K ring beside the (up to 128 KB) Q tile is twice as deep and the stream per CTA half as
 *                             wide.  Measured: +2 % at d = 256/256, 5-15 % slower at 192/64 ... 256/128: never chosen by AUTO
 *                             (DESIGN.md 6.1c).
 * The persistent plan keeps a few bytes of scheduler state per launch in device memory owned by the library: 1024 slots, each leased to
 * one launch at a time (the library records an event behind the launch and reuses the slot only after that event has completed), so
 * launches may overlap freely on any streams and host threads.  Two cases run the PER_TILE kernel instead, whatever the plan says,
 * with bit-identical results: a call on a stream that is being captured into a CUDA graph (a captured launch would hold its slot for
 * the life of the graph), and a call that finds no free slot (hundreds of persistent launches queued and unfinished).
 * Returns STREAMKL_OK, or STREAMKL_ERR_SHAPE for an unknown plan.
 */
enum { STREAMKL_FWD_AUTO = 0, STREAMKL_FWD_SINGLE = 0 /* older name of AUTO */, STREAMKL_FWD_MULTICAST = 1, STREAMKL_FWD_PAIR_MMA = 2,
       STREAMKL_FWD_PERSISTENT = 3, STREAMKL_FWD_PER_TILE = 4 };
int streamkl_set_fwd_plan(int plan);

/* Bytes of device scratch streamkl_bwd needs for this shape UNDER THE CALLING THREAD'S CURRENT MODE (O((NQ+NK)*d) at most,
 * never O(NQ*NK)): 16 B per query of packed per-query scalars, plus -- only when the one-visit strategy will run (mode FUSED,
 * or AUTO below its crossover) -- the fp32 dQ2 (and dQ1) accumulators, each region padded to 256 B. */
size_t streamkl_bwd_workspace_bytes(int B, int H, int NQ, int NK, int d1, int d2, int want_teacher_grads);

/*
 * End-to-end variants with HOST buffers (same argument meaning; `dtype` = STREAMKL_BF16 | STREAMKL_F32).
 * They take device scratch for inputs/outputs from the stream-ordered pool, copy host->device, run the kernels above,
 * copy device->host, and synchronise `stream` before returning.  Host buffers may be pageable or pinned (pinned
 * buffers are what lets the copies overlap the kernels).
 * streamkl_fwd_bwd_host runs forward then backward on the same resident inputs (one "step" of the hot path);
 * pass dQ1 = dK1 = NULL for Setting 1 only.
 */
int streamkl_fwd_host(int dtype, const void* Q1, const void* K1, const void* Q2, const void* K2,
                      int B, int H, int NQ, int NK, int d1, int d2, float c1, float c2, int causal,
                      float* kl_rows, float* lse1, float* lse2, streamkl_stream_t stream);
int streamkl_fwd_bwd_host(int dtype, const void* Q1, const void* K1, const void* Q2, const void* K2,
                          int B, int H, int NQ, int NK, int d1, int d2, float c1, float c2, int causal,
                          const float* dkl_rows, float* kl_rows, float* lse1, float* lse2,
                          void* dQ1, void* dK1, void* dQ2, void* dK2, streamkl_stream_t stream);

/*
 * The *_host entry points cut the batch into groups of whole heads (heads are independent) and overlap the upload of
 * one group and the download of another with the kernels of a third on internal streams; results are bit-identical to
 * one ungrouped call.  Their device scratch comes from the device's stream-ordered memory pool and stays cached there
 * between calls (no cudaMalloc/cudaFree per call); streamkl_host_trim() synchronises the device and returns that cached
 * memory to the driver.
 */
int streamkl_host_trim(void);

/* Number of kernels the last successful streamkl_* call on this thread launched (for launch accounting). */
int streamkl_last_launch_count(void);

/*
 * Per-kernel timing, a measurement aid (bench.py's roofline block uses it).  streamkl_profile_enable(on != 0) makes every
 * later kernel launch from the calling thread record a CUDA event on the launch stream immediately before and after
 * the kernel (on > 1 additionally creates `on` event pairs up front, so that none is created inside a timed region; events
 * are pooled and reused); streamkl_profile_collect() synchronises those events, writes up to max_records (kernel id,
 * milliseconds) pairs in launch order, forgets them and returns how many it wrote (or a negative STREAMKL_ERR_* code).
 * streamkl_kernel_name() maps a kernel id to the kernel's name (static string).  Disabled by default; when disabled
 * the launch path does not touch events at all.
 */
int streamkl_profile_enable(int on);
int streamkl_profile_collect(int max_records, int* kernel_ids, float* ms);
const char* streamkl_kernel_name(int kernel_id);

const char* streamkl_strerror(int code);
const char* streamkl_version(void);

#ifdef __cplusplus
}
#endif
#endif /* STREAMKL_H_ */
