/* scape.h — C-ABI of the SCAPE per-shard sparse optimizer step for NVIDIA B200 (sm_100a).
 *
 * What the library computes: one rank's partition of Algorithm 1 of "SCAPE: Accurate and
 * Efficient LLM Training with Extreme Sparse Communication" (arXiv 2607.01678;
 * PAPER.md:131-174), with the N data-parallel workers of the paper simulated as R gradient
 * buffers resident in one GPU's HBM and the all-reduce of Alg. 1 l.10 replaced by
 * an in-device sum over those R buffers.  Per step, in the paper's order:
 *   l.6   m~^r = beta1 m + (1-beta1) g^r + e^r
 *   l.7-8 e^r <- m~^r off the mask M_{t-1}, 0 on it
 *   l.9   b^r <- m~^r on M_{t-1}, packed: fp32 values + int32 idx
 *   l.10  b- = (1/R) sum_r b^r
 *   l.11  M_t = top-k of |m~^0| over the whole partition, used from
 *         step t+1 on (one-step delay)
 *   l.12  m <- b- (zero off the mask, Eq. 4)
 *   l.13  g^ = (b- - beta1 m_old)/(1-beta1)   (Eq. 3)
 *   l.15-17 v = beta2 m_old^2 + (1-beta2) g^^2 ; u = m/(sqrt(v)+eps);
 *         theta <- theta - lr (u + wd theta)   (AdamS, Eq. 2)
 * clip_grad (l.14) and bias correction are off by default (readings S3, S4);
 * scape_set_clip_grad / scape_set_bias_correction below switch them on.
 * Ties in the top-k go to the lower index; exactly k = N - floor(sparsity*N) entries are kept.
 * The fp32 operation order is pinned.
 *
 * All pointers are plain pointers; "device" means memory of the CUDA device that was current
 * when scape_create ran.  No call throws or aborts; failures return NULL / a negative code and
 * leave a message retrievable with scape_last_error() (thread-local).  There is no CPU
 * fallback: without a CUDA device scape_create fails.
 */
#ifndef SCAPE_H_
#define SCAPE_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct scape scape_t;

/* error codes (negative) */
#define SCAPE_OK       0
#define SCAPE_EINVAL  (-1)   /* bad argument (NULL handle, misaligned pointer, bad selector/size) */
#define SCAPE_ECUDA   (-2)   /* a CUDA runtime call or kernel launch failed                        */
#define SCAPE_ENOMEM  (-3)   /* device or host allocation failed                                   */

/* gradient element types for scape_set_grad_dtype */
#define SCAPE_GRAD_F32   0
#define SCAPE_GRAD_BF16  1

/* selectors for scape_get / scape_set / scape_count.  "LAST" = what the last completed step
 * used or produced; "NEXT" = what the coming step will use.                                      */
#define SCAPE_MOMENT        0  /* m, dense [N] f32                                    get/set      */
#define SCAPE_RESIDUAL      1  /* e^r, dense [N] f32 (argument r)                     get/set      */
#define SCAPE_MASK_NEXT     2  /* M_t: bit i%32 of word i/32, [ceil(N/32)] u32        get/set      */
#define SCAPE_MASK_LAST     3  /* M_{t-1} as used by the last step, same layout       get          */
#define SCAPE_IDX_NEXT      4  /* ascending indices of MASK_NEXT, [count] i32         get          */
#define SCAPE_IDX_LAST      5  /* ascending indices of MASK_LAST, [count] i32         get          */
#define SCAPE_PACKED        6  /* b^r of the last step, [count_last] f32 (argument r) get          */
#define SCAPE_PACKED_MEAN   7  /* b- of the last step, [count_last] f32               get          */

/* Alg. 1 "Require" line + l.1-2: create the state of one partition.
 *   shard_numel  N, number of fp32 parameters in the flattened shard, 0 < N < 2^31
 *   R            number of simulated data-parallel replicas (the paper's N workers), 1..8 (every
 *                BASELINE.json config has R <= 8; the streaming kernels are instantiated for these)
 *   sparsity     s in [0,1); k = N - floor(s*N) (evaluated in double) entries are selected
 *   beta1,beta2  in [0,1); eps >= 0; lr; wd : AdamS hyper-parameters, cast to fp32 once
 * Allocates on the current CUDA device and OWNS: m [N] (zeros), e^r [R][N] (zeros, l.2), the
 * current mask (all ones, l.1) and the next mask, index lists, packed buffers and select
 * scratch.  Returns NULL on failure (invalid argument, no device, out of memory).             */
scape_t* scape_create(int64_t shard_numel, int R, double sparsity, double beta1, double beta2,
                      double eps, double lr, double wd);

/* One pass of Alg. 1 l.4-17 over the partition.
 *   param        device, N fp32, 16-byte aligned, caller-owned, updated IN PLACE (l.17)
 *   grads        HOST array of R device pointers; grads[r] holds g^r: N elements of the type
 *                set by scape_set_grad_dtype (fp32 default), 16-byte aligned, caller-owned,
 *                never written
 *   cuda_stream  a cudaStream_t (NULL = legacy default stream)
 * All work is enqueued on cuda_stream; the call does not synchronise and allocates nothing,
 * so it can be captured into a CUDA graph -- with one rule.  The handle rotates three mask slots
 * and two packed-mean buffers from step to step and bakes their addresses, the learning rate and
 * the bias-correction factors into the launches, so a captured sequence replays correctly only if
 * it returns the rotation to where it started: capture a multiple of SCAPE_GRAPH_PERIOD (= 6)
 * consecutive steady-state steps (sparse mask in, i.e. from the third step on; constant lr, bias
 * correction off) and replay that graph any number of times; scape_step_count does not advance on
 * replay.  One step may be in flight per handle.  Advances the step counter.
 * Returns SCAPE_OK or a negative code.  On SCAPE_EINVAL nothing was enqueued and the state is
 * unchanged.  SCAPE_ECUDA means a launch or runtime call failed part-way through the step: some
 * kernels may already be enqueued, the step counter and the mask rotation have NOT advanced, and
 * the handle's contents (theta included) are undefined -- destroy the handle or reload every
 * buffer with scape_set before stepping again.                                                  */
#define SCAPE_GRAPH_PERIOD 6
int scape_step(scape_t* h, float* param, const void* const* grads, void* cuda_stream);

/* Same step with HOST buffers (end-to-end path): copies param (N fp32) and the R gradient
 * buffers host->device into handle-owned staging (allocated on first use), runs scape_step,
 * copies param back device->host, and synchronises cuda_stream before returning.  Pinned host
 * memory makes the copies asynchronous DMA; pageable memory works but is slower.
 * In steady state (sparse mask, flat top-k, no clip_grad, at least 2368 tiles of 1024 parameters)
 * the three phases are pipelined in 16 parts of whole tiles: the streaming kernel runs on sub-ranges
 * of the shard, so that theta of part i travels back while the gradients of part i + 1 travel up
 * (PCIe is full duplex), on two copy streams of the handle's own ordered by events; stage 2 follows
 * the last part.  The result is the same to the bit.
 * Bytes moved per call: h2d = 4N + R*N*sizeof(grad element), d2h = 4N.                          */
int scape_step_host(scape_t* h, float* param_host, const void* const* grads_host,
                    void* cuda_stream);

/* Synchronises the handle's device work and frees everything it owns.  NULL is a no-op.       */
void scape_destroy(scape_t* h);

/* k of reading S6; the number of completed steps t; kernels launched so far by this handle.   */
int64_t scape_k(const scape_t* h);
int64_t scape_step_count(const scape_t* h);
int64_t scape_launch_count(const scape_t* h);

/* Name of the streaming kernel the last step launched: "scape_fused_tma_kernel" (steady state:
 * bulk-copy staged) or "scape_fused_step_kernel" (register-staged: all-ones steps, dense m, small
 * or odd shapes), "" before the first step.  Static string, never NULL.                         */
const char* scape_last_kernel(const scape_t* h);

/* Number of entries of SCAPE_MASK_NEXT / SCAPE_MASK_LAST (N while the mask is all ones, else
 * k); `which` is one of those two selectors.  Negative code on error.                           */
int64_t scape_count(const scape_t* h, int which);

/* Element type of the gradient buffers passed to the following steps (S16: fp32 or bf16;
 * bf16 is widened exactly to fp32 in registers).                                               */
int scape_set_grad_dtype(scape_t* h, int dtype);

/* Optional parts of Algorithm 1 / Eq. 2 that the default configuration leaves out (DESIGN.md
 * readings S3, S4); each takes effect from the next scape_step.
 *   scape_set_lr              learning rate eta for the following steps (schedules).
 *   scape_set_bias_correction m_t/(1-beta1^t), v_t/(1-beta2^t) in l.16; t = number of
 *                             the step being taken (scape_step_count + 1).
 *   scape_set_clip_grad       l.14 clip_grad(b-bar) (PAPER.md:165; "gradient clip of 1", :279): the
 *                             reconstructed gradient g^ of the selected entries is multiplied by
 *                             max_norm / (||g^||_2 + 1e-6) when that is < 1 (the torch / Megatron
 *                             rule; the paper does not define it).  0 switches it off.  Allocates
 *                             2 N floats on first use.  With clipping on, theta of the selected
 *                             entries is updated by a second small kernel after the norm is known;
 *                             the norm is summed in double in a fixed order, so results are
 *                             reproducible run to run and agree with the oracle to ~1 ulp.
 *   scape_last_grad_norm      ||g^||_2 and the factor applied by the last step (synchronises).   */
int scape_set_lr(scape_t* h, double lr);
int scape_set_bias_correction(scape_t* h, int on);
int scape_set_clip_grad(scape_t* h, double max_norm);
int scape_last_grad_norm(scape_t* h, double* norm, double* coef, void* cuda_stream);

/* Per-layer refresh and density warm-up (readings S9, S19).
 *   scape_set_layers    PAPER.md:89 ("the top-k sparsification is performed in a per-layer style"),
 *                       :138 ("number of layers in model L"): cut the shard into n_layers layers
 *                       [offsets[l], offsets[l+1]) (HOST array of n_layers+1 entries, offsets[0] = 0,
 *                       offsets[n_layers] = shard_numel, strictly increasing; any alignment) and run
 *                       refresh_mask (l.11) inside every layer: k_l = n_l - floor(sparsity * n_l)
 *                       entries of largest |m~^0|, ties to the lower index.  compress (HOST array of
 *                       n_layers bytes, or NULL = all ones): compress[l] == 0 marks a layer that is
 *                       never sparsified (LayerNorm, RMSNorm, bias: PAPER.md:246, :279, :286): all
 *                       its entries stay selected, so it takes dense AdamS steps.  Takes effect with
 *                       the next step's refresh; masks already made stay as they are.  n_layers = 0
 *                       returns to one flat top-k.  At most SCAPE_MAX_LAYERS layers.  Synchronises
 *                       the device; allocates 32 KB per layer + 4 bytes per 128 parameters.
 *   scape_set_sparsity  sparsity of the following refreshes (density warm-up: "we use
 *                       sparsity warmup to exponentially decrease density d from 1 to 0.1 or 0.01";
 *                       the schedule is the caller's).  The mask made by step t at sparsity s_t is
 *                       used by step t+1.  Grows the packed buffers when the new masks are larger
 *                       than any before (then it synchronises the device); never shrinks them.
 *   scape_layer_k       k_l of a layer at the current sparsity (layer 0 = the whole shard when no
 *                       layers are set); scape_k is their sum.                                       */
#define SCAPE_MAX_LAYERS 4096
int scape_set_layers(scape_t* h, int n_layers, const int64_t* offsets, const uint8_t* compress);
int scape_set_sparsity(scape_t* h, double sparsity);
int64_t scape_layer_k(const scape_t* h, int layer);

/* Workers: the exchange step of Algorithm 1 across processes (not part of
 * the north-star path, which sums R replicas inside one GPU).  PAPER.md:136 ("N workers"), :155
 * (l.10: all-reduce of b), §IV-A :178 and Fig. 7 :218 ("each worker only computes a portion of the
 * top-k operations ... the new local masks from all workers are gathered").
 *   scape_set_workers   this handle is worker `rank` of `world`; every worker holds the whole
 *                       shard (theta, m, masks are identical on all of them) and its own R gradient
 *                       buffers and residuals.  layer_owner: HOST array of n_layers worker numbers
 *                       (scape_set_layers first): worker layer_owner[l] refreshes the mask of layer
 *                       l from ITS replica 0's statistic; NULL = this worker owns every layer (only
 *                       with world = 1).  The mean of l.10 becomes the sum over all R * world
 *                       replicas -- each worker's own replicas in order, then the workers' sums --
 *                       divided by R * world.  Allocates 2 N floats once.  Synchronises the device.
 *   scape_step_local    everything of a step that needs no other worker: l.6-9 for the local
 *                       replicas, the local sums of l.10, theta off the mask (l.17 with u = 0), this
 *                       worker's portion of the refresh (l.11).  Same arguments and rules as
 *                       scape_step.  clip_grad is not available in this mode (SCAPE_EINVAL).
 *   scape_exchange_buffers  what has to be summed over the workers before scape_step_apply, as
 *                       DEVICE pointers owned by the handle: `sums` = n_sums floats (the local sum of
 *                       m~^r at every selected position, in index order: the payload of l.10; an
 *                       all-reduce SUM makes it the global sum), `mask_words` = n_mask_words uint32
 *                       words of M_t in which only this worker's layers have bits (the portions are
 *                       disjoint, so an integer all-reduce SUM, or an all-gather of word-aligned
 *                       portions, completes the mask); n_mask_words = 0 when the sparsity is 0.
 *                       Valid between scape_step_local and scape_step_apply.
 *   scape_step_apply    l.10 (division), l.12-17 on the mask from the summed buffer, rank and index
 *                       list of the completed M_t; advances t.  `param` as in scape_step_local.
 * With world = 1 the pair step_local / step_apply computes exactly what scape_step computes.
 * scape_step itself refuses a handle with world > 1.  scape_set_layers / scape_set_sparsity are
 * refused between the two halves.                                                              */
int scape_set_workers(scape_t* h, int world, int rank, const int32_t* layer_owner);
int scape_step_local(scape_t* h, float* param, const void* const* grads, void* cuda_stream);
int scape_exchange_buffers(scape_t* h, float** sums, int64_t* n_sums, uint32_t** mask_words, int64_t* n_mask_words);
int scape_step_apply(scape_t* h, float* param, void* cuda_stream);

/* The exchange itself, inside the library (PAPER.md:155 l.10 "all-reduce"; §IV-A :178 "each worker
 * only computes a portion of the top-k operations"; Fig. 7 :218 "the new local masks from all
 * workers are gathered"; :236, :244 "launch the asynchronous all-gather for M_t").  Call between
 * scape_step_local and scape_step_apply, instead of exchanging scape_exchange_buffers yourself.
 *   comm        an ncclComm_t of `world` ranks whose rank numbers are the worker numbers (the
 *               caller creates it; scape_nccl_* below are there for callers without NCCL bindings).
 *               The library resolves NCCL at run time (dlopen of the libnccl.so.2 already in the
 *               process, else the system one): no link-time dependency; SCAPE_ECUDA if absent.
 *   mask_comm   a second communicator for the mask portions, or NULL.  With one, the portions travel
 *               on a stream of the handle's own, off the caller's stream: the one-step delay means
 *               M_t is not needed before the NEXT scape_step_local, which waits for it (as does
 *               every accessor).  NULL: they follow the sums on cuda_stream through `comm`.
 *   What moves: the n_sums floats (in-place all-reduce SUM), and of M_t only what each worker made:
 *               every maximal run of consecutive layers with one owner is broadcast from that owner
 *               (grouped: one all-gather-v of word ranges, not an all-reduce of all N/32 words); the
 *               at most n_layers - 1 words that hold a boundary between two owners are collected,
 *               summed (disjoint bits: SUM = OR) and put back.  scape_exchange_plan reports the plan.
 * Errors: SCAPE_EINVAL outside a split step; SCAPE_ECUDA for NCCL / CUDA failures (the split step
 * stays pending; the communicator's state is NCCL's).                                             */
int scape_step_exchange(scape_t* h, void* comm, void* mask_comm, void* cuda_stream);

/* The plan scape_step_exchange follows for the mask (a pure function of the layer offsets and
 * owners, identical on every worker).  HOST outputs, each may be NULL: *n_ranges word ranges
 * [first[i], end[i]) broadcast from worker owner[i] (arrays of capacity `cap`), and *n_shared mask
 * words shared by several owners (`shared`, capacity `cap_shared`).  Returns SCAPE_EINVAL if a
 * capacity is too small (the counts are still written).                                          */
int scape_exchange_plan(const scape_t* h, int64_t* first, int64_t* end, int32_t* owner, int cap, int* n_ranges,
                        int64_t* shared, int cap_shared, int* n_shared);

/* NCCL communicator helpers (thin forwards to ncclGetUniqueId / ncclCommInitRank / ncclCommDestroy
 * of the NCCL the library resolved).  id: HOST, SCAPE_NCCL_ID_BYTES bytes, made by one rank and
 * distributed by the caller (e.g. a torch.distributed broadcast over gloo).                      */
#define SCAPE_NCCL_ID_BYTES 128
int scape_nccl_unique_id(void* id);
int scape_nccl_comm_create(int world, int rank, const void* id, void** comm);
int scape_nccl_comm_destroy(void* comm);

/* Asynchronous mask refresh ("the delayed use of the sparse mask ... provides an
 * opportunity to ... hide" the top-k; :236 AsyncMaskRefresh).  theta, m, e^r and b are final when
 * the streaming kernel ends; M_t is not needed before the next step.  With on = 1, scape_step runs
 * stage 2 (the exact select, the rank / index list of M_t) on a stream of the handle's own, ordered
 * after the streaming kernel by an event, and returns the caller's stream as soon as that kernel is
 * enqueued: whatever the caller enqueues next (its forward / backward) overlaps the refresh.  The
 * next scape_step / scape_step_local and every accessor make their stream wait for the refresh
 * first; scape_join_refresh does so explicitly.  A step captured into a CUDA graph always runs the
 * refresh in-stream, and a capture cannot wait for work enqueued outside it: call
 * scape_join_refresh on the stream the graph will be launched on before capturing (SCAPE_EINVAL
 * otherwise).  Default off.  scape_step_exchange with a mask_comm uses the same stream.   */
int scape_set_async_refresh(scape_t* h, int on);
int scape_join_refresh(scape_t* h, void* cuda_stream);

/* Algorithm 2, parameter side (Eq. 6 :207-211).  With
 * Megatron-LM's distributed optimizer only the OWNER of a partition holds its updated parameters
 * w'; before the next forward pass the others need them.  Eq. 6: after the update of step t,
 * theta differs from (1 - eta lambda) theta only on M_{t-1}, the mask that update used -- so only
 * those k values travel (Alg. 2 l.2-3) and every worker decays the rest itself from its full FP32
 * copy (l.4, "Use FP32 w to compute untransmitted params", :231-232).  Both calls work on the mask
 * the handle's LAST completed step used (SCAPE_MASK_LAST / SCAPE_IDX_LAST; all N entries after the
 * first step, whose mask is all ones), enqueue one kernel on cuda_stream and return without
 * synchronising.  The all-gather between them is the caller's.  DESIGN.md readings S21-S23.
 *   scape_param_pack    l.2  w~ <- w'[M_{t-1}]: out[j] = param[idx_last[first + j]], 0 <= j < count,
 *                       ascending index order (the order of the sparse buffer), as fp32
 *                       (SCAPE_PARAM_F32) or rounded to nearest even to bf16 (SCAPE_PARAM_BF16).
 *                       param: DEVICE, N fp32 (the array scape_step updates); out: DEVICE, count
 *                       elements, caller-owned.  [first, first + count) must lie inside
 *                       [0, scape_count(h, SCAPE_MASK_LAST)): a worker that owns a range of the
 *                       sparse buffer packs just that range.
 *   scape_param_apply   l.3-4 on a copy of the shard that did NOT take the update: w (DEVICE, N
 *                       fp32, 16-byte aligned, the full FP32 copy, updated IN PLACE) gets
 *                       w[i] = payload[j] on the mask (payload: DEVICE, scape_count(MASK_LAST)
 *                       elements of `dtype` in index order, i.e. the gathered w~) and
 *                       w[i] = fma(-eta, lambda w[i], w[i]) off it -- Alg. 1 l.17 with u = 0, the
 *                       arithmetic the owner itself applies there, so that with an fp32 payload w
 *                       equals the owner's parameters bit for bit ((1 - eta lambda) w of Eq. 6
 *                       differs from it by at most 1 ulp); eta is the learning rate the last step
 *                       applied.  w_hat (DEVICE, N bf16, 8-byte aligned, or NULL): the compute
 *                       copy, w_hat[i] = bf16(w[i]) (round to nearest even) for every i.
 * SCAPE_EINVAL before the first step, during a split step, for a bad range, dtype or alignment.   */
#define SCAPE_PARAM_F32   0
#define SCAPE_PARAM_BF16  1
int scape_param_pack(scape_t* h, const float* param, int64_t first, int64_t count, void* out, int dtype,
                     void* cuda_stream);
int scape_param_apply(scape_t* h, float* w, void* w_hat, const void* payload, int dtype, void* cuda_stream);

/* Mask bit pack / unpack, stand-alone (no handle).  PAPER.md:250-252: "we convert the masks from INT8
 * to 1-bit values and pack 8 mask values into one byte" (the paper's Triton kernels, K1 of SURVEY.md
 * §2).  The packed form is the one SCAPE_MASK_NEXT / SCAPE_MASK_LAST and scape_exchange_buffers use:
 * bit i % 32 of little-endian word i / 32, bits at positions >= n zero.
 *   scape_mask_pack    mask_bytes: DEVICE, n bytes, non-zero = selected; words: DEVICE,
 *                      ceil(n / 32) uint32, completely overwritten.
 *   scape_mask_unpack  the inverse: writes n bytes of 0 / 1.
 * Both enqueue one kernel on cuda_stream of the CURRENT device and return without synchronising.
 * Buffers are caller-owned.  n = 0 is a no-op.  SCAPE_EINVAL for n < 0, NULL or misaligned words.  */
int scape_mask_pack(const uint8_t* mask_bytes, int64_t n, uint32_t* words, void* cuda_stream);
int scape_mask_unpack(const uint32_t* words, int64_t n, uint8_t* mask_bytes, void* cuda_stream);

/* Ordered compaction of a bit mask WITHOUT any allocation (stage 4's index half, PAPER.md:144, :154:
 * "indices into the flattened shard"), stand-alone (no handle), for callers that
 * cannot call cudaMalloc: code under CUDA graph capture, tight serving loops, harnesses that forbid
 * it.  The scratch of the scan (the look-back state of one CTA per 131,072 bits) is a file-scope
 * __device__ array of the library, 33 KB, held by every GPU that loads the library until the
 * process exits; hence the limit n <= SCAPE_STATIC_MAX_BITS.
 *   mask_words  DEVICE, ceil(n / 32) uint32, 16-byte aligned: bit i % 32 of word i / 32 (the layout of
 *               SCAPE_MASK_NEXT / scape_mask_pack); bits at positions >= n are ignored.  Read only.
 *   idx_out     DEVICE, idx_cap int32: the positions of the set bits in ascending order (what
 *               SCAPE_IDX_NEXT holds for the same mask).  Entries beyond idx_cap are dropped; *count_out
 *               still counts them.  May be NULL when idx_cap = 0 (count only).
 *   count_out   DEVICE, one uint32: the number of set bits among the first n.
 * Enqueues two small memsets of the scratch and one kernel on cuda_stream of the CURRENT device (the one
 * that owns the buffers) and returns without synchronising.  Calls cudaMalloc / cudaFree never; the first
 * call on a device resolves the array's address (cudaGetSymbolAddress), later calls only launch.
 * All calls on one device share the scratch array: calls that may OVERLAP on the GPU (different
 * streams without an ordering between them) race and give wrong results; calls ordered on one stream,
 * or by events, are fine.  n = 0 sets *count_out = 0.
 * SCAPE_EINVAL for n < 0, n > SCAPE_STATIC_MAX_BITS (message names the limit), idx_cap < 0, NULL or
 * misaligned pointers; SCAPE_ECUDA when a CUDA call fails.                                          */
#define SCAPE_STATIC_MAX_BITS 536870912LL   /* 2^29 */
int scape_mask_indices_static(const uint32_t* mask_words, int64_t n, int32_t* idx_out, int64_t idx_cap,
                              uint32_t* count_out, void* cuda_stream);

/* How rank128 + the index list are made from the bits of a new mask: 0 = by shard size (default:
 * one pass with a chained scan up to 2^26 parameters, three kernels above), 1 = always the single
 * pass, 2 = always the three kernels.  Both forms give identical results; for tests.            */
int scape_set_compaction(scape_t* h, int form);

/* Option: also materialise b^r on steps whose mask is all ones (step 1, or sparsity 0), where
 * the packed buffer would be R*N floats.  Off by default: on such steps SCAPE_PACKED is then
 * unavailable (SCAPE_EINVAL) and SCAPE_PACKED_MEAN equals SCAPE_MOMENT.  Allocates R*N floats
 * when switched on.  For tests.                                                                */
int scape_set_keep_dense_pack(scape_t* h, int on);

/* State accessors (tests, checkpoint/resume, the "identical state each step" loader).  `buf`
 * may be a host or a device pointer (unified addressing); `bytes` must equal the size of the
 * selected object; `r` is the replica for SCAPE_RESIDUAL / SCAPE_PACKED and ignored otherwise.
 * Both calls synchronise `cuda_stream` before returning.  Not part of the timed path.
 * scape_set(SCAPE_MASK_NEXT) accepts a mask with at most as many set bits as the largest mask so
 * far (scape_k at creation, grown by scape_set_sparsity / scape_set_layers), or with all N bits set;
 * bits at positions >= N are ignored; a mask with more bits is refused (SCAPE_EINVAL) and the
 * handle keeps the mask it had.  scape_set is refused between scape_step_local and
 * scape_step_apply.                                                                            */
int scape_get(scape_t* h, int what, int r, void* buf, size_t bytes, void* cuda_stream);
int scape_set(scape_t* h, int what, int r, const void* buf, size_t bytes, void* cuda_stream);
int scape_set_step_count(scape_t* h, int64_t t);

/* How often the stage-2 select could use the candidate list gathered by the fused pass (the
 * threshold predicted from the previous step bracketed the true one: `fast`) and how often it
 * fell back to radix passes over the whole partition (`general`; always the case on all-ones
 * steps).  With layers set the counts are per layer and step.  Both routes are exact.
 * Synchronises cuda_stream.                                     */
int scape_select_stats(scape_t* h, int64_t* fast, int64_t* general, void* cuda_stream);
/* Of the steps scape_select_stats counts as "general", how many the recovery pass saved from re-reading
 * every key three to five times: a bracket taken from a sampled histogram, ONE classification pass over
 * the keys, then the candidate route (a missed prediction, the first step).  HOST output.            */
int scape_select_recovered(scape_t* h, int64_t* recovered, void* cuda_stream);

/* Diagnostics of the last step's select (not graded): out8 = {bracket held (0/1), entries above
 * the bracket, candidates, half-width of the next bracket in ln units, ln of the exact threshold,
 * ln of the threshold predicted for the next step, candidate capacity, candidate segments}.
 * Synchronises cuda_stream.                                                                      */
int scape_select_debug(scape_t* h, double* out8, void* cuda_stream);

/* Optional timing, for bench.py's roofline: while switched on, every scape_step also records
 * three CUDA events on its stream (before the fused streaming kernel of stages 1,3-6, after it,
 * and after the stage-2 select), at most 64 steps between reads without a host wait.
 * scape_profile(h, on) resets the totals.  scape_profile_read waits for the recorded events and
 * returns the summed milliseconds of the fused kernel and of the select stage and the number of
 * steps they cover (any pointer may be NULL).                                                   */
int scape_profile(scape_t* h, int on);
int scape_profile_read(scape_t* h, double* fused_ms, double* select_ms, int64_t* steps);

/* Message of the last failure on the calling thread ("" if none).  Never NULL.                 */
const char* scape_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* SCAPE_H_ */
