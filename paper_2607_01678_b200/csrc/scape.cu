// scape.cu — host side of libscape.so: the C-ABI of include/scape.h, the handle, and the
// stream-ordered launch sequence of one SCAPE step (Algorithm 1, :131-174).
// No CPU fallback exists: every stage runs in the kernels of scape_kernels.cuh.
#include "../../include/scape.h"

#include <dlfcn.h>

#include <algorithm>
#include <functional>
#include <mutex>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "scape_select_kernels.cuh"

// kernel lookups exported by the instantiation units (scape_fused_inst.cu)
namespace scapek {
#define SCAPE_DECL_INST(tag)                                                               \
  const void* fused_step_kernel_##tag(int R, bool dense, bool msparse, bool clipt);        \
  const void* fused_tma_kernel_##tag(int R, bool clipt, bool rkview, uint32_t* tile_bytes);
SCAPE_DECL_INST(f32_lo)
SCAPE_DECL_INST(f32_hi)
SCAPE_DECL_INST(bf16_lo)
SCAPE_DECL_INST(bf16_hi)
#undef SCAPE_DECL_INST
}  // namespace scapek

using namespace scapek;

static_assert(scapek::SCAPE_MAX_LAYERS_K == SCAPE_MAX_LAYERS, "layer-end table of the select kernels");

namespace {

thread_local char g_err[512] = "";

int fail(int code, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof g_err, fmt, ap);
  va_end(ap);
  return code;
}

#define CU_TRY(expr)                                                                         \
  do {                                                                                       \
    cudaError_t _e = (expr);                                                                 \
    if (_e != cudaSuccess) return fail(SCAPE_ECUDA, "%s: %s", #expr, cudaGetErrorString(_e)); \
  } while (0)

// shards of up to this many 1024-chunk blocks (2^26 parameters) compact their masks in one pass
constexpr int kSinglePassCompactBlocks = 512;

struct MaskSlot {
  uint32_t* bits = nullptr;   // [n_words]
  uint2* rank = nullptr;      // [n_chunks] {set bits before the chunk, running popcounts of its words}
  uint32_t* pre = nullptr;    // [8 * n_tiles] the second half of `rank` on its own (zero past n_chunks)
  uint32_t* trank = nullptr;  // [n_tiles + 1] set bits before every tile of 8 chunks; last entry: all of them
  int32_t* idx = nullptr;     // [k]   (not materialised while all_ones)
  int64_t count = 0;
  bool all_ones = false;
  bool valid = false;
};

// one streaming-kernel instantiation as this handle launches it
struct FusedCfg {
  const void* fn = nullptr;   // kernel address (scape_fused_inst.cu); nullptr: the instantiation does not exist
  int bps = 0;                // resident CTAs per SM the grid is sized for
  int stages = 0;             // staged kernel: ring depth
  uint32_t tile = 0;          // staged kernel: bytes per stage
  size_t smem = 0;            // dynamic shared memory per CTA
};

struct DeviceGuard {
  int prev = -1;
  bool ok = true;
  explicit DeviceGuard(int dev) {
    if (cudaGetDevice(&prev) != cudaSuccess) { ok = false; return; }
    if (prev != dev && cudaSetDevice(dev) != cudaSuccess) ok = false;
  }
  ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

}  // namespace

struct scape {
  int64_t N = 0, Npad = 0, n_chunks = 0, n_words = 0, k = 0;
  int R = 0, dev = 0, n_sm = 148, grad_dtype = SCAPE_GRAD_F32;
  int64_t t = 0, launches = 0;
  float b1, b2, eps, lr, wd, c1, c2;
  float lr_last = 0.0f;        // learning rate the last completed step applied (scape_param_apply decays with it)

  float* m = nullptr;          // [Npad]
  float* e = nullptr;          // [R][Npad]
  // three mask slots rotate: `use` = M_{t-1}, the mask the coming step uses (SCAPE_MASK_NEXT);
  // `last` = the mask the last step used (SCAPE_MASK_LAST; a sparsely stored m is addressed
  // through it); `build` = where the coming step writes M_t
  MaskSlot slot[3];
  int use = 0, last = 1, build = 2;
  float* packed = nullptr;     // [R][packed_stride]
  int64_t packed_stride = 0;
  float* pm[2] = {nullptr, nullptr};   // packed means b- [packed_stride], alternating
  int pm_last = 0;             // pm[pm_last] = b- of the last sparse step
  const char* last_kernel = "";   // name of the streaming kernel the last step launched
  // optional parts of Alg. 1 (off by default: readings S3, S4)
  bool bias_correction = false;
  double beta1_d = 0.0, beta2_d = 0.0, clip_max_norm = 0.0;
  float* ghat = nullptr;       // [Npad] clip mode: g^ of the selected entries (packed; dense steps use all N)
  float* vm = nullptr;         // [Npad] clip mode: beta2 * m_old^2 of the selected entries
  double* sumsq = nullptr;     // [max_seg] clip mode: per-warp partial sums of g^^2
  ClipState* clip_state = nullptr;
  // launch configuration of the streaming kernels for this handle's R on this handle's device
  // (prepare_kernels): [gradient type][variant][clip_grad instantiation]
  FusedCfg cfg_step[2][3][2];
  FusedCfg cfg_tma[2][2][2];   // ... [table view: 0 pre + trank (flat top-k), 1 rk (per-layer refresh)]
  bool m_sparse = false;       // m_{t-1} lives in pm[pm_last] addressed through slot[last]; h->m is stale
  float* dense_pack = nullptr;    // optional [R][Npad]
  bool last_dense = false;

  SelState* sel = nullptr;
  unsigned long long* cls = nullptr;    // [kClsCap] small list of the radix select
  unsigned long long* cand = nullptr;   // [cand_cap] candidate composite keys of the fused select
  int64_t cand_cap = 0;
  uint32_t* seg_count = nullptr;  // [max_seg]
  uint32_t* seg_above = nullptr;  // [max_seg]
  int max_seg = 0;
  uint32_t* ghist = nullptr;      // [kBins]
  uint32_t* block_sum = nullptr;  // [n_compact_blocks]
  uint32_t* warp_pre = nullptr;   // [n_compact_blocks * 32] set bits before each group of 32 chunks inside its block of 1024
  uint32_t* total = nullptr;      // [2]: number of set bits, ticket of mask_compact_kernel
  unsigned long long* scan_state = nullptr;   // [n_compact_blocks] look-back state of mask_compact_kernel
  uint32_t compact_epoch = 0;
  int compact_impl = 0;           // 1 single pass (small shards), 0 count / scan / rank (scape_set_compaction)
  int n_compact_blocks = 0;
  int n_seg = 0;                  // segments (= warps) of the last fused launch
  int n_slots = 0;                // warps of the last streaming launch (clip-mode partial sums)
  uint32_t seg_cap = 0;

  // per-layer refresh (scape_set_layers) and per-step sparsity (scape_set_sparsity)
  double sparsity = 0.0;          // sparsity of the coming refreshes
  int n_layers = 0;               // 0 = one flat top-k over the shard
  std::vector<int64_t> lay_off;   // host copy [n_layers + 1]
  std::vector<uint8_t> lay_compress;
  LayerState* layers = nullptr;   // [n_layers]
  LayerCtl* lctl = nullptr;
  uint32_t* chunk_layer = nullptr;   // [n_chunks]
  uint32_t* lhist = nullptr;      // [n_layers][kBins]
  int4* items = nullptr;
  int n_items = 0;

  // workers (scape_set_workers): this handle is worker `rank` of `world`; the step is split into
  // scape_step_local / [all-reduce of the exchange buffers] / scape_step_apply
  int world = 1, rank = 0;
  std::vector<uint8_t> lay_skip;  // host copy: layers whose mask another worker makes
  // the mask part of scape_step_exchange (a pure function of the layer offsets and owners, the same
  // on every worker): word ranges broadcast from their owner + the words two owners share
  std::vector<int64_t> xr_first, xr_end, x_shared;
  std::vector<int32_t> xr_owner;
  uint32_t* x_shared_idx = nullptr;   // [x_shared.size()] device copy of the shared word numbers
  uint32_t* x_shared_buf = nullptr;   // [x_shared.size()] their values, summed over the workers
  bool pending_mask_on_side = false;  // the mask portions travel on `side`: scape_step_apply compacts there

  // asynchronous refresh (scape_set_async_refresh) and the mask exchange with its own communicator:
  // a stream of the handle's own, ordered against the caller's stream by two events
  bool async_refresh = false;
  cudaStream_t side = nullptr;
  cudaEvent_t ev_main = nullptr, ev_side = nullptr;
  bool side_used = false;         // ev_side has been recorded: the caller's stream must wait for it
  bool side_dirty = false;        // ... and no stream has waited for it since (a capture cannot wait: it needs this false)

  // The flat select + compaction is 14-16 small dependent launches whose arguments only depend on the
  // mask rotation (which slots), the route forced or not, k and the segment layout: each distinct
  // sequence is captured once into a CUDA graph and replayed with one launch afterwards (shards under
  // ~2^23 parameters are launch-bound: pr1 0.113 -> see DESIGN.md ms per step)
  struct SelGraph { long long key[11]; cudaGraphExec_t exec; int launches; };
  std::vector<SelGraph> sel_graphs;
  cudaStream_t cap_stream = nullptr;
  bool use_sel_graphs = true;
  bool fused_hist_made = false;   // the last streaming launch added the candidates' first-digit histogram to ghist

  bool pending = false;           // step_local has run, step_apply has not
  bool pending_need_select = false;
  int pending_pm_out = 0;
  float pending_bc1 = 1.0f, pending_bc2 = 1.0f, pending_lr = 0.0f;

  // optional per-step CUDA-event timing of the fused kernel and of the select stage
  bool prof_on = false;
  static constexpr int kProfRing = 64;
  cudaEvent_t prof_ev[kProfRing][3] = {};
  bool prof_have_events = false;
  int prof_pending = 0;              // steps recorded since the last drain
  double prof_fused_ms = 0.0, prof_select_ms = 0.0;
  int64_t prof_steps = 0;

  int32_t* iota_scratch = nullptr;   // scape_get(SCAPE_IDX_*) of an all-ones mask

  // scape_step_host staging and pipeline (upload / download streams, one event pair per part)
  static constexpr int kHostParts = 16;
  cudaStream_t up = nullptr, down = nullptr;
  cudaEvent_t ev_up[kHostParts] = {}, ev_cmp[kHostParts] = {}, ev_host = nullptr;
  float* st_param = nullptr;
  void* st_grad[kMaxR] = {};
  size_t st_grad_bytes = 0;
};

namespace {

int grid_for(const scape* h, int64_t n_chunks, int warps_per_block, int blocks_per_sm) {
  int64_t need = (n_chunks + warps_per_block - 1) / warps_per_block;
  int64_t cap = (int64_t)h->n_sm * blocks_per_sm;
  if (need < 1) need = 1;
  return (int)(need < cap ? need : cap);
}

// ---- the handle's own stream (asynchronous refresh, mask exchange) --------------------------------
int ensure_side(scape* h) {
  if (h->side) return SCAPE_OK;
  // highest priority: the refresh is a chain of small dependent kernels; at default priority its blocks
  // queue behind whatever grid the caller has in flight and the chain stretches over the caller's whole
  // forward / backward (measured: no overlap at all), at high priority they take the SM slots as they free up
  int prio_lo = 0, prio_hi = 0;
  CU_TRY(cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi));
  CU_TRY(cudaStreamCreateWithPriority(&h->side, cudaStreamNonBlocking, prio_hi));
  CU_TRY(cudaEventCreateWithFlags(&h->ev_main, cudaEventDisableTiming));
  CU_TRY(cudaEventCreateWithFlags(&h->ev_side, cudaEventDisableTiming));
  return SCAPE_OK;
}

bool is_capturing(cudaStream_t st) {
  cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
  if (cudaStreamIsCapturing(st, &cs) != cudaSuccess) { cudaGetLastError(); return false; }
  return cs != cudaStreamCaptureStatusNone;
}

// Everything the handle enqueued on its own stream happens before what `st` gets from now on.  A
// capturing stream cannot wait for an event recorded outside the capture: there the work must be over.
int join_side(scape* h, cudaStream_t st) {
  if (!h->side_used) return SCAPE_OK;
  if (is_capturing(st)) {
    // (no event query either: inside a global-mode capture it invalidates the capture)
    if (h->side_dirty)
      return fail(SCAPE_EINVAL, "work on the handle's own stream has not been joined: scape_join_refresh on the stream the graph "
                                "will be launched on (or a device synchronisation) before capturing");
    return SCAPE_OK;
  }
  CU_TRY(cudaStreamWaitEvent(st, h->ev_side, 0));
  h->side_dirty = false;
  return SCAPE_OK;
}

// side <- after everything enqueued on st so far
int fork_side(scape* h, cudaStream_t st) {
  int rc = ensure_side(h);
  if (rc) return rc;
  CU_TRY(cudaEventRecord(h->ev_main, st));
  CU_TRY(cudaStreamWaitEvent(h->side, h->ev_main, 0));
  return SCAPE_OK;
}

int mark_side(scape* h) {
  CU_TRY(cudaEventRecord(h->ev_side, h->side));
  h->side_used = true;
  h->side_dirty = true;
  return SCAPE_OK;
}

// ---- NCCL, resolved at run time (no link-time dependency; the paper's own data plane) ----
struct NcclId { char internal[SCAPE_NCCL_ID_BYTES]; };
struct NcclApi {
  void* lib = nullptr;
  int (*AllReduce)(const void*, void*, size_t, int, int, void*, cudaStream_t) = nullptr;
  int (*Broadcast)(const void*, void*, size_t, int, int, void*, cudaStream_t) = nullptr;
  int (*GroupStart)() = nullptr;
  int (*GroupEnd)() = nullptr;
  const char* (*GetErrorString)(int) = nullptr;
  int (*GetUniqueId)(NcclId*) = nullptr;
  int (*CommInitRank)(void**, int, NcclId, int) = nullptr;
  int (*CommDestroy)(void*) = nullptr;
};
constexpr int kNcclFloat32 = 7, kNcclUint32 = 3, kNcclSum = 0;      // nccl.h: ncclDataType_t / ncclRedOp_t

const NcclApi* nccl() {
  static NcclApi api;
  static bool tried = false;
  if (tried) return api.lib ? &api : nullptr;
  tried = true;
  // the copy already in the process (torch loads its own) wins over the system's
  void* lib = dlopen("libnccl.so.2", RTLD_NOW | RTLD_NOLOAD | RTLD_GLOBAL);
  if (!lib) lib = dlopen("libnccl.so.2", RTLD_NOW | RTLD_GLOBAL);
  if (!lib) lib = dlopen("libnccl.so", RTLD_NOW | RTLD_GLOBAL);
  if (!lib) return nullptr;
  bool ok = true;
  auto sym = [&](const char* name) { void* f = dlsym(lib, name); if (!f) ok = false; return f; };
  api.AllReduce = (decltype(api.AllReduce))sym("ncclAllReduce");
  api.Broadcast = (decltype(api.Broadcast))sym("ncclBroadcast");
  api.GroupStart = (decltype(api.GroupStart))sym("ncclGroupStart");
  api.GroupEnd = (decltype(api.GroupEnd))sym("ncclGroupEnd");
  api.GetErrorString = (decltype(api.GetErrorString))sym("ncclGetErrorString");
  api.GetUniqueId = (decltype(api.GetUniqueId))sym("ncclGetUniqueId");
  api.CommInitRank = (decltype(api.CommInitRank))sym("ncclCommInitRank");
  api.CommDestroy = (decltype(api.CommDestroy))sym("ncclCommDestroy");
  if (!ok) return nullptr;
  api.lib = lib;
  return &api;
}

#define NCCL_TRY(api, expr)                                                                       \
  do {                                                                                            \
    int _r = (expr);                                                                              \
    if (_r != 0) return fail(SCAPE_ECUDA, "%s: %s", #expr, (api)->GetErrorString(_r));            \
  } while (0)

// Mask part of the exchange: every maximal run of consecutive layers with one owner becomes a word
// range [first, end) that only this owner writes; a word that holds a boundary between two runs is
// shared.  offsets == nullptr (no layers): one run, owner 0.
void build_exchange_plan(scape* h, const int32_t* layer_owner) {
  h->xr_first.clear(); h->xr_end.clear(); h->xr_owner.clear(); h->x_shared.clear();
  const int64_t n_words = (h->N + 31) / 32;
  if (h->n_layers == 0 || !layer_owner) {
    h->xr_first.push_back(0); h->xr_end.push_back(n_words); h->xr_owner.push_back(0);
    return;
  }
  int l = 0;
  while (l < h->n_layers) {
    int e = l + 1;
    while (e < h->n_layers && layer_owner[e] == layer_owner[l]) ++e;
    const int64_t a = h->lay_off[l], b = h->lay_off[e];
    const int64_t w0 = (a + 31) / 32, w1 = b == h->N ? n_words : b / 32;
    if (w1 > w0) { h->xr_first.push_back(w0); h->xr_end.push_back(w1); h->xr_owner.push_back(layer_owner[l]); }
    if (a % 32 != 0 && (h->x_shared.empty() || h->x_shared.back() != a / 32)) h->x_shared.push_back(a / 32);
    l = e;
  }
}

// The streaming kernels are instantiated in scape_fused_inst.cu (one translation unit per gradient
// type and range of R); their launch configuration is resolved ONCE PER HANDLE in
// prepare_kernels(), under the handle's device: occupancy and the opt-in to more than 48 KB of
// dynamic shared memory are per device, and handles of several devices may live in one process.
const void* step_kernel(int dtype, int R, bool dense, bool msparse, bool clipt) {
  const void* f = dtype == SCAPE_GRAD_BF16 ? fused_step_kernel_bf16_lo(R, dense, msparse, clipt)
                                           : fused_step_kernel_f32_lo(R, dense, msparse, clipt);
  if (!f) f = dtype == SCAPE_GRAD_BF16 ? fused_step_kernel_bf16_hi(R, dense, msparse, clipt)
                                       : fused_step_kernel_f32_hi(R, dense, msparse, clipt);
  return f;
}

const void* tma_kernel(int dtype, int R, bool clipt, bool rkview, uint32_t* tile) {
  const void* f = dtype == SCAPE_GRAD_BF16 ? fused_tma_kernel_bf16_lo(R, clipt, rkview, tile) : fused_tma_kernel_f32_lo(R, clipt, rkview, tile);
  if (!f) f = dtype == SCAPE_GRAD_BF16 ? fused_tma_kernel_bf16_hi(R, clipt, rkview, tile) : fused_tma_kernel_f32_hi(R, clipt, rkview, tile);
  return f;
}

int prepare_kernels(scape* h) {
  for (int dt = 0; dt < 2; ++dt)
    for (int clipt = 0; clipt < 2; ++clipt) {
      for (int v = 0; v < 3; ++v) {          // 0 all-ones mask | 1 sparse mask, dense m in | 2 sparse mask, sparse m in
        FusedCfg& c = h->cfg_step[dt][v][clipt];
        c.fn = step_kernel(dt, h->R, v == 0, v == 2, clipt != 0);
        if (!c.fn) return fail(SCAPE_EINVAL, "no streaming kernel for R = %d", h->R);
        // sparse variants: per-warp scratch of the on-mask arithmetic + candidate ring (dynamic shared memory)
        c.smem = step_smem_bytes(h->R, v == 0);
        if (c.smem > 48u * 1024u) CU_TRY(cudaFuncSetAttribute(c.fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c.smem));
        int occ = 0;
        CU_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, c.fn, 256, c.smem));
        c.bps = occ > 0 ? (occ > 8 ? 8 : occ) : 1;
      }
      // Staged kernel: two CTAs (16 consumer warps) per SM with >= 3 stages each, or not at all
      // (tma_can_launch in scape_kernels.cuh); as many stages as fit, at most kTmaMaxStages.
      for (int view = 0; view < 2; ++view) {
      FusedCfg& c = h->cfg_tma[dt][clipt][view];
      c.fn = tma_kernel(dt, h->R, clipt != 0, view != 0, &c.tile);
      if (c.fn) {
        if (view == 0) {       // flat form: barriers + as many stages as fit
          const int s2 = (int)((kSmemPerSm / 2u - 1024u - kTmaBarrierBytes) / c.tile);
          c.stages = s2 > kTmaMaxStages ? kTmaMaxStages : s2;
          c.smem = kTmaBarrierBytes + (size_t)c.stages * c.tile;
        } else {               // grouped form: + two mask buffers (a group's mask words, by bulk copy); at most kTmaGroup
                               // stages (the producer's reuse rule for the mask buffers needs n_stages <= kTmaGroup)
          const uint32_t mb = tma_mb_bytes<true>();
          const int s2 = (int)((kSmemPerSm / 2u - 1024u - kTmagBarrierBytes - 2u * mb) / c.tile);
          c.stages = s2 > kTmaGroup ? kTmaGroup : s2;
          c.smem = kTmagBarrierBytes + 2u * mb + (size_t)c.stages * c.tile;
        }
        c.bps = 2;
        CU_TRY(cudaFuncSetAttribute(c.fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c.smem));
      }
      }
    }
  return SCAPE_OK;
}

void set_segments(scape* h, StepParams& p, int n_seg) {
  // one candidate segment per warp of this step's launch(es)
  if (n_seg > h->max_seg) n_seg = h->max_seg;
  h->n_seg = n_seg;
  h->n_slots = n_seg;
  int64_t cap = (h->cand_cap / h->n_seg) & ~(int64_t)15;
  if (cap > 0x7FFFFFF0) cap = 0x7FFFFFF0;
  h->seg_cap = (uint32_t)cap;
  p.seg_cap = h->seg_cap;
}

// variants: all-ones mask (dense m in and out) | sparse mask, dense m in | sparse mask, sparse m in
// part / n_parts: the launch covers the part-th of n_parts ranges of the shard (scape_step_host's pipeline;
// boundaries at whole tiles); every part uses its own block of candidate segments.  1 part = the whole shard.
int launch_fused(scape* h, StepParams& p, bool dense, bool msparse, cudaStream_t st, int part = 0, int n_parts = 1) {
  const int64_t tiles_all = (p.n_chunks + 7) / 8;
  p.c_begin = (uint32_t)(8 * (tiles_all * part / n_parts));
  p.c_end = part + 1 == n_parts ? (uint32_t)p.n_chunks : (uint32_t)(8 * (tiles_all * (part + 1) / n_parts));
  const int64_t range_chunks = (int64_t)p.c_end - (int64_t)p.c_begin;
  const int dt = h->grad_dtype == SCAPE_GRAD_BF16 ? 1 : 0, clipt = p.clip ? 1 : 0;   // the clip_grad variant is its own instantiation
  // The staged kernel wins when there are enough bytes per parameter to be HBM-bound (R >= 3);
  // with one or two replicas the step is issue-bound and the register-staged kernel's higher
  // occupancy (40 warps/SM vs 16 consumer warps) is worth more (measured at N = 2^28, 99 %:
  // R = 1: 1.49 vs 2.02 ms, R = 2: 1.95 vs 2.08 ms, R = 4: 2.94 vs 2.72 ms).
  const int view = h->n_layers > 0 ? 1 : 0;          // per-layer refresh: the grouped form (consumer-bound there)
  const FusedCfg& ct = h->cfg_tma[dt][clipt][view];
  if (!dense && msparse && ct.fn && h->R >= 3 && p.N / kTmaTile >= (int64_t)h->n_sm * n_parts && (view == 0 || n_parts == 1)) {
    const int64_t n_tiles = n_parts == 1 ? p.N / kTmaTile : std::min<int64_t>(p.N / kTmaTile, p.c_end / 8) - p.c_begin / 8;
    const int64_t n_units = view ? (n_tiles + kTmaGroup - 1) / kTmaGroup : n_tiles;   // grouped: a CTA takes groups of kTmaGroup consecutive tiles
    int64_t grid = (int64_t)h->n_sm * ct.bps;
    if (grid > n_units) grid = n_units;
    if (part == 0) set_segments(h, p, (n_parts == 1 ? (int)grid : h->n_sm * ct.bps) * kTmaConsumerWarps * n_parts);
    p.fused_hist = nullptr; h->fused_hist_made = false;
    p.seg_cap = h->seg_cap;
    p.seg_base = (uint32_t)(part * h->n_sm * ct.bps * kTmaConsumerWarps);
    int stages = ct.stages;
    void* args[] = {(void*)&p, (void*)&stages};
    CU_TRY(cudaLaunchKernel(ct.fn, dim3((unsigned)grid), dim3(kTmaThreads), args, ct.smem, st));
    h->last_kernel = "scape_fused_tma_kernel";
    h->launches++;
    return SCAPE_OK;
  }
  const FusedCfg& c = h->cfg_step[dt][dense ? 0 : msparse ? 2 : 1][clipt];
  const int grid = grid_for(h, range_chunks, 8, c.bps);
  if (part == 0) set_segments(h, p, (n_parts == 1 ? grid : h->n_sm * c.bps) * 8 * n_parts);
  // flat top-k: the kernel histograms the candidates' first radix digit as it flushes them (sel_decide_kernel)
  // (not on small shards: zeroing and merging 1024 counters per CTA costs a launch-bound kernel more than the pass it saves)
  h->fused_hist_made = !dense && h->n_layers == 0 && h->k < h->N && h->N >= ((int64_t)1 << 24);
  p.fused_hist = h->fused_hist_made ? h->ghist : nullptr;
  p.seg_cap = h->seg_cap;
  p.seg_base = (uint32_t)(part * h->n_sm * c.bps * 8);
  void* args[] = {(void*)&p};
  CU_TRY(cudaLaunchKernel(c.fn, dim3((unsigned)grid), dim3(256), args, c.smem, st));
  h->last_kernel = "scape_fused_step_kernel";
  h->launches++;
  return SCAPE_OK;
}

// dense view of m in h->m when it is stored sparsely (accessors; all-ones step after sparse ones)
int materialise_dense_m(scape* h, cudaStream_t st) {
  if (!h->m_sparse) return SCAPE_OK;
  const MaskSlot& s = h->slot[h->last];
  CU_TRY(cudaMemsetAsync(h->m, 0, sizeof(float) * h->Npad, st));
  if (s.count > 0) {
    scatter_packed_kernel<<<1024, 256, 0, st>>>(h->m, s.idx, h->pm[h->pm_last], s.count);
    h->launches++;
    CU_TRY(cudaGetLastError());
  }
  return SCAPE_OK;
}

static_assert((int64_t)kScanMaxPer * 1024 * kCompactChunksPerBlock * 128 >= ((int64_t)1 << 31), "mask_scan_blocks_kernel: one block scans every block sum of a shard");
// rank128 (+ idx when idx != nullptr) of slot.bits; leaves the bit count in *h->total
int compact_mask(scape* h, MaskSlot& s, bool want_idx, cudaStream_t st) {
  const int nb = h->n_compact_blocks;
  if (h->compact_impl == 1) {       // single pass (chained scan with look-back)
    h->compact_epoch = (h->compact_epoch + 1u) & 0x3FFFFFFFu;
    mask_compact_kernel<<<nb, 1024, 0, st>>>(s.bits, h->n_chunks, h->scan_state, h->total, h->compact_epoch, s.rank, s.pre, s.trank,
                                            want_idx ? s.idx : nullptr, h->packed_stride);
    h->launches += 1;
    CU_TRY(cudaGetLastError());
    return SCAPE_OK;
  }
  mask_block_count_kernel<<<nb, kCountThreads, 0, st>>>(s.bits, h->n_chunks, h->block_sum, h->warp_pre);
  mask_scan_blocks_kernel<<<1, 1024, 0, st>>>(h->block_sum, nb, h->total);
  mask_rank_idx_kernel<<<nb * (kCompactChunksPerBlock / (kRankIdxThreads * kRankIdxGroups)), kRankIdxThreads, 0, st>>>(
                                            s.bits, h->n_chunks, h->block_sum, h->warp_pre, s.rank, s.pre, s.trank, want_idx ? s.idx : nullptr,
                                            h->packed_stride);
  h->launches += 3;
  CU_TRY(cudaGetLastError());
  return SCAPE_OK;
}

// Stage 2 (Alg. 1 l.11): exact top-k of |m~^0| -> nxt.bits / rank / idx.  When the fused pass ran
// with a predicted bracket (sparse step) the radix select works on its candidate list if the
// bracket held; otherwise (or on all-ones steps: force_general) on every key of the partition.
int run_select_direct(scape* h, const MaskSlot& cur, MaskSlot& nxt, bool force_general, cudaStream_t st, bool compact) {
  KeySrc src;
  src.e0 = h->e;
  src.cur_bits = cur.all_ones ? nullptr : cur.bits;
  src.cur_rk = cur.all_ones ? nullptr : cur.rank;
  src.packed0 = h->packed;
  src.N = h->N;
  src.n_chunks = h->n_chunks;
  CandList cl;
  cl.cls = h->cls; cl.cand = h->cand; cl.seg_count = h->seg_count; cl.seg_above = h->seg_above;
  cl.seg_cap = h->seg_cap; cl.n_seg = force_general ? 0 : h->n_seg;
  // the recovery pass's own segment layout: one segment per warp of its launch -- 5 CTAs per SM on large shards, one
  // warp per 8 chunks on small ones (so that a segment keeps room for its share of the candidates)
  cl.rec_n_seg = (int)std::min<int64_t>((int64_t)h->n_sm * 5 * 8, std::max<int64_t>(8, (h->n_chunks / 8 + 7) / 8 * 8));
  cl.rec_seg_cap = (uint32_t)std::min<int64_t>((h->cand_cap / cl.rec_n_seg) & ~(int64_t)15, 0x7FFFFFF0);
  const int grid = grid_for(h, h->n_chunks, 8, 6);
  sel_decide_kernel<<<1, 1024, 0, st>>>(h->sel, h->ghist, cl, (long long)h->k, force_general ? 1 : 0,
                                        (!force_general && h->fused_hist_made) ? 1 : 0);
  // a missed bracket (or none: all-ones step): bracket from a sampled histogram, one classification pass, then the
  // candidate route; all four return at once when the predicted bracket held (sel_sample_kernel)
  sel_sample_kernel<<<grid, 256, 0, st>>>(src, h->sel, h->ghist);
  sel_sample_pick_kernel<<<1, 1024, 0, st>>>(h->sel, h->ghist, (long long)h->k, (long long)h->N);
  sel_classify_kernel<<<cl.rec_n_seg / 8, 256, 0, st>>>(src, cl, h->sel, h->cand, h->seg_count, h->seg_above, nxt.bits);
  sel_decide2_kernel<<<1, 1024, 0, st>>>(h->sel, cl, (long long)h->k);
  h->launches += 5;
  // 64 undecided bits at most, 13 per pass; the kernels take the digit position from the state
  // and return at once when nothing is left to decide (fast route: 4 passes are typical)
  for (int p = 0; p < kSelPasses; ++p) {
    sel_hist_kernel<<<grid, 256, 0, st>>>(src, cl, h->sel, h->ghist, nxt.bits);
    sel_pick_kernel<<<1, 1024, 0, st>>>(h->sel, h->ghist);
    h->launches += 2;
  }
  sel_finish_kernel<<<grid, 256, 0, st>>>(src, cl, h->sel, nxt.bits);
  h->launches++;
  CU_TRY(cudaGetLastError());
  if (!compact) return SCAPE_OK;
  int rc = compact_mask(h, nxt, true, st);
  if (rc) return rc;
  nxt.count = h->k;
  nxt.all_ones = false;
  nxt.valid = true;
  return SCAPE_OK;
}

void drop_sel_graphs(scape* h) {
  for (auto& g : h->sel_graphs) cudaGraphExecDestroy(g.exec);
  h->sel_graphs.clear();
}

// run_select_direct through a cached CUDA graph (see scape::SelGraph).  Falls back to the direct launches
// inside a caller's capture, and whenever capturing or instantiating fails.
int run_select_layered_direct(scape* h, const MaskSlot& cur, MaskSlot& nxt, bool force_general, cudaStream_t st, bool compact);

// layered: the per-layer select (its 25 launches as one graph: 0.1 ms of dependency latency less on the headline shard);
// its kernels take the layer tables' addresses, the item count and the sparsity by value (scape_set_layers drops the graphs)
int run_select(scape* h, const MaskSlot& cur, MaskSlot& nxt, bool force_general, cudaStream_t st, bool compact = true, bool layered = false) {
  auto direct = [layered](scape* h_, const MaskSlot& cur_, MaskSlot& nxt_, bool fg, cudaStream_t st_, bool compact_) {
    return layered ? run_select_layered_direct(h_, cur_, nxt_, fg, st_, compact_) : run_select_direct(h_, cur_, nxt_, fg, st_, compact_);
  };
  if (!h->use_sel_graphs || is_capturing(st)) return direct(h, cur, nxt, force_general, st, compact);
  long long sparsity_bits = 0;
  std::memcpy(&sparsity_bits, &h->sparsity, sizeof(double));
  long long key[11] = {(long long)(&cur - h->slot), (long long)(&nxt - h->slot), (force_general ? 1 : 0) | (cur.all_ones ? 2 : 0), compact ? 1 : 0,
                       (long long)h->n_seg, (long long)h->seg_cap, (long long)h->k, (long long)h->compact_impl | (h->fused_hist_made ? 256 : 0),
                       layered ? 1 : 0, (long long)h->n_layers, layered ? sparsity_bits : 0};
  for (auto& g : h->sel_graphs)
    if (std::memcmp(g.key, key, sizeof key) == 0) {
      CU_TRY(cudaGraphLaunch(g.exec, st));
      h->launches += g.launches;
      if (compact) { nxt.count = h->k; nxt.all_ones = false; nxt.valid = true; }
      return SCAPE_OK;
    }
  if (!h->cap_stream && cudaStreamCreateWithFlags(&h->cap_stream, cudaStreamNonBlocking) != cudaSuccess) {
    cudaGetLastError(); h->cap_stream = nullptr;
    return direct(h, cur, nxt, force_general, st, compact);
  }
  if (h->sel_graphs.size() >= 24) drop_sel_graphs(h);          // (a density schedule changes k every step)
  const int64_t l0 = h->launches;
  cudaGraph_t graph = nullptr;
  cudaGraphExec_t exec = nullptr;
  if (cudaStreamBeginCapture(h->cap_stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
    cudaGetLastError();
    return direct(h, cur, nxt, force_general, st, compact);
  }
  const int rc = direct(h, cur, nxt, force_general, h->cap_stream, compact);
  const cudaError_t ce = cudaStreamEndCapture(h->cap_stream, &graph);
  const int n_launch = (int)(h->launches - l0);
  h->launches = l0;
  if (rc != SCAPE_OK || ce != cudaSuccess || !graph || cudaGraphInstantiate(&exec, graph, 0) != cudaSuccess) {
    cudaGetLastError();
    if (graph) cudaGraphDestroy(graph);
    h->use_sel_graphs = false;                                   // not available here: direct launches from now on
    return direct(h, cur, nxt, force_general, st, compact);
  }
  cudaGraphDestroy(graph);
  scape::SelGraph g;
  std::memcpy(g.key, key, sizeof key);
  g.exec = exec; g.launches = n_launch;
  h->sel_graphs.push_back(g);
  CU_TRY(cudaGraphLaunch(exec, st));
  h->launches += n_launch;
  return SCAPE_OK;
}

// Storage whose size follows the number of selected entries: index lists, packed b^r, the two
// packed means, the candidate list.  Grows (never shrinks) so that masks of up to K entries fit;
// live contents are kept.  Synchronises the device when it has to reallocate.  Masks with all N
// bits set need none of it.
int ensure_capacity(scape* h, int64_t K) {
  if (K >= h->N) return SCAPE_OK;
  const int64_t stride = (K + 31) / 32 * 32;
  if (stride > h->packed_stride) {
    CU_TRY(cudaDeviceSynchronize());
    drop_sel_graphs(h);                                          // the graphs hold the old buffers' addresses
    const int64_t old = h->packed_stride;
    auto grow = [&](void** p, size_t elem, int64_t rows) -> bool {
      void* q = nullptr;
      if (cudaMalloc(&q, elem * (size_t)stride * rows) != cudaSuccess) { cudaGetLastError(); return false; }
      if (cudaMemset(q, 0, elem * (size_t)stride * rows) != cudaSuccess) { cudaFree(q); return false; }
      if (*p && old > 0)
        for (int64_t r = 0; r < rows; ++r)
          if (cudaMemcpy((char*)q + elem * (size_t)stride * r, (char*)*p + elem * (size_t)old * r, elem * (size_t)old,
                         cudaMemcpyDeviceToDevice) != cudaSuccess) { cudaFree(q); return false; }
      cudaFree(*p);
      *p = q;
      return true;
    };
    bool ok = true;
    for (auto& s : h->slot) ok = ok && grow((void**)&s.idx, sizeof(int32_t), 1);
    ok = ok && grow((void**)&h->pm[0], sizeof(float), 1) && grow((void**)&h->pm[1], sizeof(float), 1);
    ok = ok && grow((void**)&h->packed, sizeof(float), h->R);
    if (!ok) return fail(SCAPE_ENOMEM, "device allocation failed (packed buffers for %lld selected entries)", (long long)K);
    h->packed_stride = stride;
  }
  {
    // candidates of the fused select: room for 4k keys (a bracket of +-3 % around the threshold
    // holds ~0.8k: error feedback piles residuals up just below it), at least N/8, at most N/2.
    // Grows with the largest K seen (density warm-up from the sparse side); its contents only live
    // inside a step, so nothing is copied.  Never shrinks.
    int64_t cc = 4 * K;
    if (cc < h->N / 8) cc = h->N / 8;      // very sparse masks / transients: keep room per warp segment
    if (cc > h->N / 2) cc = h->N / 2;
    if (cc < 65536) cc = 65536;
    if (!h->cls && cudaMalloc((void**)&h->cls, sizeof(unsigned long long) * (size_t)kClsCap) != cudaSuccess) {
      cudaGetLastError(); h->cls = nullptr;
      return fail(SCAPE_ENOMEM, "device allocation failed (small list of the select)");
    }
    if (cc > h->cand_cap) {
      drop_sel_graphs(h);
      if (h->cand) { CU_TRY(cudaDeviceSynchronize()); cudaFree(h->cand); h->cand = nullptr; h->cand_cap = 0; }
      if (cudaMalloc((void**)&h->cand, sizeof(unsigned long long) * (size_t)cc) != cudaSuccess) {
        cudaGetLastError(); h->cand = nullptr;
        return fail(SCAPE_ENOMEM, "device allocation failed (candidate list)");
      }
      h->cand_cap = cc;
    }
  }
  return SCAPE_OK;
}

// entries the refresh selects at sparsity s: reading S6, inside every layer when layers are set
int64_t total_k(const scape* h, double s) {
  if (h->n_layers == 0) return h->N - (int64_t)std::floor(s * (double)h->N);
  int64_t K = 0;
  for (int l = 0; l < h->n_layers; ++l) {
    const int64_t n = h->lay_off[l + 1] - h->lay_off[l];
    K += h->lay_compress[l] ? n - (int64_t)std::floor(s * (double)n) : n;
  }
  return K;
}

// Stage 2 with layers: the same exact select inside every layer at once.
int run_select_layered(scape* h, const MaskSlot& cur, MaskSlot& nxt, bool force_general, cudaStream_t st, bool compact = true) {
  return run_select(h, cur, nxt, force_general, st, compact, /*layered=*/true);
}

int run_select_layered_direct(scape* h, const MaskSlot& cur, MaskSlot& nxt, bool force_general, cudaStream_t st, bool compact) {
  KeySrc src;
  src.e0 = h->e;
  src.cur_bits = cur.all_ones ? nullptr : cur.bits;
  src.cur_rk = cur.all_ones ? nullptr : cur.rank;
  src.packed0 = h->packed;
  src.N = h->N;
  src.n_chunks = h->n_chunks;
  CandList cl;
  cl.cls = h->cls; cl.cand = h->cand; cl.seg_count = h->seg_count; cl.seg_above = h->seg_above;
  cl.seg_cap = h->seg_cap; cl.n_seg = force_general ? 0 : h->n_seg;
  LayerWork w;
  w.chunk_layer = h->chunk_layer; w.layers = h->layers; w.n_layers = h->n_layers; w.ctl = h->lctl;
  w.hist = h->lhist; w.items = h->items; w.n_items = h->n_items;
  const int grid_c = h->n_sm * 6;      // 6 CTAs of 256 threads per SM (the 32 KB layer-end table bounds it)
  int grid_f = h->n_sm * 6; if (grid_f > h->n_items) grid_f = h->n_items;
  lsel_decide_kernel<<<1, 1024, 0, st>>>(w, cl, h->sparsity, force_general ? 1 : 0);
  h->launches++;
  // 5 digits at most, plus one round for layers whose bracket turns out (first pick) to have
  // missed and that restart on the general route; kernels with nothing to do return at once
  for (int round = 0; round < kSelPasses + 1; ++round) {
    if (!force_general) { lsel_hist_cand_kernel<<<grid_c, 256, 0, st>>>(w, cl, nxt.bits); h->launches++; }
    lsel_hist_full_kernel<<<grid_f, 256, 0, st>>>(src, w);
    lsel_pick_kernel<<<h->n_layers, kLayerPickThreads, 0, st>>>(w);
    h->launches += 2;
  }
  lsel_finish_full_kernel<<<grid_f, 256, 0, st>>>(src, w, nxt.bits);
  h->launches++;
  if (!force_general) { lsel_finish_cand_kernel<<<grid_c, 256, 0, st>>>(w, cl, nxt.bits); h->launches++; }
  CU_TRY(cudaGetLastError());
  if (!compact) return SCAPE_OK;          // workers: the other workers' bits are still missing (scape_step_apply)
  int rc = compact_mask(h, nxt, true, st);
  if (rc) return rc;
  nxt.count = h->k;
  nxt.all_ones = false;
  nxt.valid = true;
  return SCAPE_OK;
}

// fold the recorded event pairs into the running totals (synchronises on the events)
int prof_drain(scape* h) {
  for (int i = 0; i < h->prof_pending; ++i) {
    float a = 0.f, b = 0.f;
    CU_TRY(cudaEventSynchronize(h->prof_ev[i][2]));
    CU_TRY(cudaEventElapsedTime(&a, h->prof_ev[i][0], h->prof_ev[i][1]));
    CU_TRY(cudaEventElapsedTime(&b, h->prof_ev[i][1], h->prof_ev[i][2]));
    h->prof_fused_ms += a; h->prof_select_ms += b; h->prof_steps += 1;
  }
  h->prof_pending = 0;
  return SCAPE_OK;
}

bool finite_all(std::initializer_list<double> v) {
  for (double x : v) if (!std::isfinite(x)) return false;
  return true;
}

void free_all(scape* h) {
  cudaFree(h->m); cudaFree(h->e);
  for (auto& s : h->slot) { cudaFree(s.bits); cudaFree(s.rank); cudaFree(s.pre); cudaFree(s.trank); cudaFree(s.idx); }
  cudaFree(h->packed); cudaFree(h->pm[0]); cudaFree(h->pm[1]); cudaFree(h->dense_pack);
  cudaFree(h->sel); cudaFree(h->cand); cudaFree(h->cls); cudaFree(h->seg_count); cudaFree(h->seg_above); cudaFree(h->ghist); cudaFree(h->block_sum); cudaFree(h->warp_pre); cudaFree(h->total); cudaFree(h->scan_state);
  cudaFree(h->ghat); cudaFree(h->vm); cudaFree(h->sumsq); cudaFree(h->clip_state);
  cudaFree(h->layers); cudaFree(h->lctl); cudaFree(h->chunk_layer); cudaFree(h->lhist); cudaFree(h->items);
  cudaFree(h->st_param); cudaFree(h->iota_scratch);
  cudaFree(h->x_shared_idx); cudaFree(h->x_shared_buf);
  if (h->side) { cudaStreamDestroy(h->side); cudaEventDestroy(h->ev_main); cudaEventDestroy(h->ev_side); }
  for (auto& g : h->sel_graphs) cudaGraphExecDestroy(g.exec);
  h->sel_graphs.clear();
  if (h->cap_stream) cudaStreamDestroy(h->cap_stream);
  if (h->up) {
    cudaStreamDestroy(h->up); cudaStreamDestroy(h->down); cudaEventDestroy(h->ev_host);
    for (auto& e : h->ev_up) cudaEventDestroy(e);
    for (auto& e : h->ev_cmp) cudaEventDestroy(e);
  }
  for (auto& g : h->st_grad) cudaFree(g);
  if (h->prof_have_events)
    for (auto& row : h->prof_ev) for (auto& ev : row) cudaEventDestroy(ev);
}

}  // namespace

extern "C" const char* scape_last_error(void) { return g_err; }

extern "C" scape_t* scape_create(int64_t N, int R, double sparsity, double beta1, double beta2, double eps,
                                 double lr, double wd) {
  g_err[0] = 0;
  if (!finite_all({sparsity, beta1, beta2, eps, lr, wd})) { fail(SCAPE_EINVAL, "non-finite argument"); return nullptr; }
  if (N <= 0 || N >= ((int64_t)1 << 31)) { fail(SCAPE_EINVAL, "shard_numel must be in (0, 2^31)"); return nullptr; }
  if (R < 1 || R > kMaxR) { fail(SCAPE_EINVAL, "R must be in [1, %d]", kMaxR); return nullptr; }
  if (!(sparsity >= 0.0 && sparsity < 1.0)) { fail(SCAPE_EINVAL, "sparsity must be in [0, 1)"); return nullptr; }
  if (!(beta1 >= 0.0 && beta1 < 1.0) || !(beta2 >= 0.0 && beta2 < 1.0)) { fail(SCAPE_EINVAL, "beta must be in [0, 1)"); return nullptr; }
  if (eps < 0.0) { fail(SCAPE_EINVAL, "eps must be >= 0"); return nullptr; }

  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) { fail(SCAPE_ECUDA, "no CUDA device (there is no CPU fallback)"); cudaGetLastError(); return nullptr; }
  scape* h = new (std::nothrow) scape();
  if (!h) { fail(SCAPE_ENOMEM, "host allocation failed"); return nullptr; }
  h->dev = dev;
  cudaDeviceGetAttribute(&h->n_sm, cudaDevAttrMultiProcessorCount, dev);
  h->N = N; h->R = R;
  h->Npad = (N + kChunk - 1) / kChunk * kChunk;
  h->n_chunks = h->Npad / kChunk;
  h->n_words = h->Npad / 32;
  h->k = N - (int64_t)std::floor(sparsity * (double)N);          // reading S6
  // hyper-parameters are cast to fp32 once; 1 - beta is evaluated in fp32
  h->b1 = (float)beta1; h->b2 = (float)beta2; h->eps = (float)eps; h->lr = (float)lr; h->wd = (float)wd;
  h->c1 = 1.0f - h->b1; h->c2 = 1.0f - h->b2;
  h->beta1_d = beta1; h->beta2_d = beta2;
  h->n_compact_blocks = (int)((h->n_chunks + kCompactChunksPerBlock - 1) / kCompactChunksPerBlock);
  h->sparsity = sparsity;
  h->max_seg = h->n_sm * 8 * 8 * scape::kHostParts;          // 8 CTAs x 8 warps per SM, times the parts of scape_step_host's pipeline

  bool ok = true;
  auto alloc = [&](void** p, size_t bytes, bool zero) {
    if (!ok) return;
    if (cudaMalloc(p, bytes ? bytes : 16) != cudaSuccess) { ok = false; *p = nullptr; return; }
    if (zero && cudaMemset(*p, 0, bytes ? bytes : 16) != cudaSuccess) ok = false;
  };
  alloc((void**)&h->m, sizeof(float) * h->Npad, true);                       // S5: m_0 = 0
  alloc((void**)&h->e, sizeof(float) * h->Npad * R, true);                   // l.2: e_0 = 0
  for (auto& s : h->slot) {
    // (padded with zeros to whole groups of kTmaGroup tiles = 32 chunks: the staged kernel fetches a group's
    // mask words and table entries with fixed-size bulk copies)
    const size_t chunks_pad = (size_t)((h->n_chunks + 8 * kTmaGroup - 1) / (8 * kTmaGroup)) * (8 * kTmaGroup);
    alloc((void**)&s.bits, sizeof(uint32_t) * 4 * chunks_pad, true);
    alloc((void**)&s.rank, sizeof(uint2) * chunks_pad, true);
    alloc((void**)&s.pre, sizeof(uint32_t) * chunks_pad, true);
    alloc((void**)&s.trank, sizeof(uint32_t) * (chunks_pad / 8 + kTmaGroup), true);
  }
  alloc((void**)&h->sel, sizeof(SelState), true);
  alloc((void**)&h->seg_count, sizeof(uint32_t) * h->max_seg, true);
  alloc((void**)&h->seg_above, sizeof(uint32_t) * h->max_seg, true);
  if (ok && ensure_capacity(h, h->k) != SCAPE_OK) ok = false;                // index lists, packed buffers, candidates
  alloc((void**)&h->ghist, sizeof(uint32_t) * kBins, true);
  alloc((void**)&h->block_sum, sizeof(uint32_t) * (h->n_compact_blocks + 1), true);
  alloc((void**)&h->warp_pre, sizeof(uint32_t) * 32 * (h->n_compact_blocks + 1), true);
  alloc((void**)&h->total, 2 * sizeof(uint32_t), true);
  alloc((void**)&h->scan_state, sizeof(unsigned long long) * (h->n_compact_blocks + 1), true);
  // measured: the single pass wins while launch count matters (pr1: select stage 99 -> 94 us) and loses on
  // large shards, where 13.5 k CTAs wait on one another's prefixes (headline: 0.44 -> 0.50 ms)
  h->compact_impl = h->n_compact_blocks <= kSinglePassCompactBlocks ? 1 : 0;
  if (!ok) {
    fail(SCAPE_ENOMEM, "device allocation failed: %s", cudaGetErrorString(cudaGetLastError()));
    free_all(h); delete h; return nullptr;
  }
  {
    SelState init{};
    init.br.delta = 0.5f;                     // no history yet: wide first bracket
    init.br.lo_key = init.br.hi_key = 0xFFFFFFFFu;   // nothing predicted: the first sparse step decides "general"
    if (cudaMemcpy(h->sel, &init, sizeof init, cudaMemcpyHostToDevice) != cudaSuccess) {
      fail(SCAPE_ECUDA, "create: cannot initialise the select state");
      free_all(h); delete h; return nullptr;
    }
  }
  if (prepare_kernels(h) != SCAPE_OK) { free_all(h); delete h; return nullptr; }
  h->slot[0].all_ones = true;                                                // l.1: M_0 = 1
  h->slot[0].count = N;
  h->slot[0].valid = true;
  h->use = 0; h->last = 1; h->build = 2;
  if (cudaDeviceSynchronize() != cudaSuccess) { fail(SCAPE_ECUDA, "create: sync failed"); free_all(h); delete h; return nullptr; }
  return h;
}

extern "C" void scape_destroy(scape_t* h) {
  if (!h) return;
  DeviceGuard g(h->dev);
  cudaDeviceSynchronize();
  free_all(h);
  delete h;
}

extern "C" int64_t scape_k(const scape_t* h) { return h ? h->k : SCAPE_EINVAL; }
extern "C" int64_t scape_step_count(const scape_t* h) { return h ? h->t : SCAPE_EINVAL; }
extern "C" int64_t scape_launch_count(const scape_t* h) { return h ? h->launches : SCAPE_EINVAL; }
extern "C" const char* scape_last_kernel(const scape_t* h) { return h ? h->last_kernel : ""; }

extern "C" int64_t scape_count(const scape_t* h, int which) {
  if (!h) return fail(SCAPE_EINVAL, "NULL handle");
  if (which == SCAPE_MASK_NEXT) return h->slot[h->use].count;
  if (which == SCAPE_MASK_LAST) {
    if (!h->slot[h->last].valid || h->t == 0) return fail(SCAPE_EINVAL, "no step has run yet");
    return h->slot[h->last].count;
  }
  return fail(SCAPE_EINVAL, "scape_count: bad selector %d", which);
}

extern "C" int scape_set_grad_dtype(scape_t* h, int dtype) {
  if (!h) return fail(SCAPE_EINVAL, "NULL handle");
  if (dtype != SCAPE_GRAD_F32 && dtype != SCAPE_GRAD_BF16) return fail(SCAPE_EINVAL, "unknown grad dtype %d", dtype);
  if (dtype != h->grad_dtype) {            // staging buffers are sized by dtype
    for (auto& g : h->st_grad) { cudaFree(g); g = nullptr; }
    h->st_grad_bytes = 0;
  }
  h->grad_dtype = dtype;
  return SCAPE_OK;
}

extern "C" int scape_set_keep_dense_pack(scape_t* h, int on) {
  if (!h) return fail(SCAPE_EINVAL, "NULL handle");
  DeviceGuard g(h->dev);
  if (on && !h->dense_pack) {
    if (cudaMalloc((void**)&h->dense_pack, sizeof(float) * h->Npad * h->R) != cudaSuccess) {
      h->dense_pack = nullptr; cudaGetLastError();
      return fail(SCAPE_ENOMEM, "keep_dense_pack: allocation of R*N floats failed");
    }
  } else if (!on && h->dense_pack) {
    cudaDeviceSynchronize();
    cudaFree(h->dense_pack);
    h->dense_pack = nullptr;
  }
  return SCAPE_OK;
}

extern "C" int scape_set_compaction(scape_t* h, int form) {
  if (!h) return fail(SCAPE_EINVAL, "NULL handle");
  if (form < 0 || form > 2) return fail(SCAPE_EINVAL, "form must be 0 (by size), 1 (single pass) or 2 (three kernels)");
  h->compact_impl = form == 0 ? (h->n_compact_blocks <= kSinglePassCompactBlocks ? 1 : 0) : form == 1 ? 1 : 0;
  return SCAPE_OK;
}

extern "C" int scape_set_lr(scape_t* h, double lr) {
  if (!h || !std::isfinite(lr)) return fail(SCAPE_EINVAL, "bad argument");
  h->lr = (float)lr;
  return SCAPE_OK;
}

extern "C" int scape_set_bias_correction(scape_t* h, int on) {
  if (!h) return fail(SCAPE_EINVAL, "NULL handle");
  h->bias_correction = on != 0;
  return SCAPE_OK;
}

extern "C" int scape_set_clip_grad(scape_t* h, double max_norm) {
  if (!h || !(max_norm >= 0.0) || !std::isfinite(max_norm)) return fail(SCAPE_EINVAL, "max_norm must be finite and >= 0");
  DeviceGuard g(h->dev);
  if (max_norm > 0.0 && (!h->ghat || !h->sumsq)) {
    const int slots = h->n_sm * 8 * 8;
    bool ok = (h->ghat || cudaMalloc((void**)&h->ghat, sizeof(float) * h->Npad) == cudaSuccess) &&
              (h->vm || cudaMalloc((void**)&h->vm, sizeof(float) * h->Npad) == cudaSuccess) &&
              (h->sumsq || cudaMalloc((void**)&h->sumsq, sizeof(double) * slots) == cudaSuccess) &&
              (h->clip_state || cudaMalloc((void**)&h->clip_state, sizeof(ClipState)) == cudaSuccess);
    if (!ok) {
      cudaGetLastError();
      cudaFree(h->ghat); cudaFree(h->vm); cudaFree(h->sumsq); cudaFree(h->clip_state);
      h->ghat = h->vm = nullptr; h->sumsq = nullptr; h->clip_state = nullptr;
      return fail(SCAPE_ENOMEM, "clip_grad: allocation of 2 N floats failed");
    }
    cudaMemset(h->clip_state, 0, sizeof(ClipState));
  }
  h->clip_max_norm = max_norm;
  return SCAPE_OK;
}

extern "C" int scape_set_sparsity(scape_t* h, double sparsity) {
  if (!h) return fail(SCAPE_EINVAL, "NULL handle");
  if (!(sparsity >= 0.0 && sparsity < 1.0)) return fail(SCAPE_EINVAL, "sparsity must be in [0, 1)");
  if (h->pending) return fail(SCAPE_EINVAL, "a split step is in flight");
  DeviceGuard g(h->dev);
  const int64_t K = total_k(h, sparsity);
  int rc = ensure_capacity(h, K);
  if (rc) return rc;
  h->sparsity = sparsity;
  h->k = K;
  return SCAPE_OK;
}

extern "C" int scape_set_layers(scape_t* h, int n_layers, const int64_t* offsets, const uint8_t* compress) {
  if (!h) return fail(SCAPE_EINVAL, "NULL handle");
  if (h->pending) return fail(SCAPE_EINVAL, "a split step is in flight");
  if (h->world > 1) return fail(SCAPE_EINVAL, "this handle is one of %d workers: scape_set_workers(h, 1, 0, NULL) before changing the layers", h->world);
  DeviceGuard g(h->dev);
  CU_TRY(cudaDeviceSynchronize());
  drop_sel_graphs(h);                        // the per-layer graphs hold the layer tables' addresses and the item count
  if (n_layers == 0) {                       // back to one flat top-k
    h->n_layers = 0; h->lay_off.clear(); h->lay_compress.clear();
    h->k = total_k(h, h->sparsity);
    return ensure_capacity(h, h->k);
  }
  if (n_layers < 0 || n_layers > SCAPE_MAX_LAYERS) return fail(SCAPE_EINVAL, "n_layers must be in [0, %d]", SCAPE_MAX_LAYERS);
  if (!offsets) return fail(SCAPE_EINVAL, "NULL offsets");
  if (offsets[0] != 0 || offsets[n_layers] != h->N) return fail(SCAPE_EINVAL, "offsets must run from 0 to shard_numel");
  for (int l = 0; l < n_layers; ++l)
    if (offsets[l + 1] <= offsets[l]) return fail(SCAPE_EINVAL, "offsets must be strictly increasing (layer %d is empty)", l);

  // host tables: layer of every chunk's first entry (bit 31: the chunk holds several layers), and
  // work items of at most kItemChunks chunks that never cross a layer boundary
  std::vector<uint32_t> cl((size_t)h->n_chunks);
  std::vector<int4> items;
  std::vector<LayerState> ls((size_t)n_layers);
  {
    int l = 0;
    for (int64_t c = 0; c < h->n_chunks; ++c) {
      const int64_t a = c * kChunk, b = std::min<int64_t>(a + kChunk, h->N);
      while (offsets[l + 1] <= a) ++l;
      cl[(size_t)c] = (uint32_t)l | (offsets[l + 1] < b ? 0x80000000u : 0u);
    }
  }
  for (int l = 0; l < n_layers; ++l) {
    LayerState& S = ls[(size_t)l];
    std::memset(&S, 0, sizeof S);
    S.begin = offsets[l]; S.end = offsets[l + 1];
    S.compress = compress ? (compress[l] != 0) : 1;
    S.br.delta = 0.5f;
    // nothing predicted yet for a compressed layer; every key of an uncompressed one is "above"
    S.br.lo_key = S.br.hi_key = S.compress ? 0xFFFFFFFFu : 0u;
    const int64_t c0 = S.begin / kChunk, c1 = (S.end + kChunk - 1) / kChunk;
    for (int64_t c = c0; c < c1; c += kItemChunks)
      items.push_back(make_int4(l, (int)c, (int)std::min<int64_t>(c + kItemChunks, c1), 0));
  }
  cudaFree(h->layers); cudaFree(h->lctl); cudaFree(h->chunk_layer); cudaFree(h->lhist); cudaFree(h->items);
  h->layers = nullptr; h->lctl = nullptr; h->chunk_layer = nullptr; h->lhist = nullptr; h->items = nullptr;
  h->n_layers = 0;
  bool ok = cudaMalloc((void**)&h->layers, sizeof(LayerState) * ls.size()) == cudaSuccess &&
            cudaMalloc((void**)&h->lctl, sizeof(LayerCtl)) == cudaSuccess &&
            cudaMalloc((void**)&h->chunk_layer, sizeof(uint32_t) * cl.size()) == cudaSuccess &&
            cudaMalloc((void**)&h->lhist, sizeof(uint32_t) * (size_t)kBins * ls.size()) == cudaSuccess &&
            cudaMalloc((void**)&h->items, sizeof(int4) * items.size()) == cudaSuccess;
  ok = ok && cudaMemcpy(h->layers, ls.data(), sizeof(LayerState) * ls.size(), cudaMemcpyHostToDevice) == cudaSuccess &&
       cudaMemset(h->lctl, 0, sizeof(LayerCtl)) == cudaSuccess &&
       cudaMemcpy(h->chunk_layer, cl.data(), sizeof(uint32_t) * cl.size(), cudaMemcpyHostToDevice) == cudaSuccess &&
       cudaMemset(h->lhist, 0, sizeof(uint32_t) * (size_t)kBins * ls.size()) == cudaSuccess &&
       cudaMemcpy(h->items, items.data(), sizeof(int4) * items.size(), cudaMemcpyHostToDevice) == cudaSuccess;
  if (!ok) {
    cudaGetLastError();
    cudaFree(h->layers); cudaFree(h->lctl); cudaFree(h->chunk_layer); cudaFree(h->lhist); cudaFree(h->items);
    h->layers = nullptr; h->lctl = nullptr; h->chunk_layer = nullptr; h->lhist = nullptr; h->items = nullptr;
    h->lay_off.clear(); h->lay_compress.clear();
    h->k = total_k(h, h->sparsity);
    return fail(SCAPE_ENOMEM, "set_layers: device allocation failed");
  }
  h->n_layers = n_layers;
  h->n_items = (int)items.size();
  h->lay_off.assign(offsets, offsets + n_layers + 1);
  h->lay_compress.resize((size_t)n_layers);
  for (int l = 0; l < n_layers; ++l) h->lay_compress[(size_t)l] = ls[(size_t)l].compress ? 1 : 0;
  h->k = total_k(h, h->sparsity);
  return ensure_capacity(h, h->k);
}

extern "C" int64_t scape_layer_k(const scape_t* h, int layer) {
  if (!h) return fail(SCAPE_EINVAL, "NULL handle");
  if (h->n_layers == 0) return layer == 0 ? h->k : fail(SCAPE_EINVAL, "no layers are set");
  if (layer < 0 || layer >= h->n_layers) return fail(SCAPE_EINVAL, "layer %d out of range", layer);
  const int64_t n = h->lay_off[layer + 1] - h->lay_off[layer];
  return h->lay_compress[layer] ? n - (int64_t)std::floor(h->sparsity * (double)n) : n;
}

extern "C" int scape_last_grad_norm(scape_t* h, double* norm, double* coef, void* cuda_stream) {
  if (!h) return fail(SCAPE_EINVAL, "NULL handle");
  if (!h->clip_state) return fail(SCAPE_EINVAL, "clip_grad has never been switched on");
  DeviceGuard g(h->dev);
  ClipState cs{};
  CU_TRY(cudaMemcpyAsync(&cs, h->clip_state, sizeof cs, cudaMemcpyDeviceToHost, (cudaStream_t)cuda_stream));
  CU_TRY(cudaStreamSynchronize((cudaStream_t)cuda_stream));
  if (norm) *norm = cs.norm;
  if (coef) *coef = (double)cs.coef;
  return SCAPE_OK;
}

extern "C" int scape_set_step_count(scape_t* h, int64_t t) {
  if (!h || t < 0) return fail(SCAPE_EINVAL, "bad argument");
  h->t = t;
  return SCAPE_OK;
}

namespace {

// Elements [first, end) of part i of n: the same boundaries launch_fused uses (whole tiles of 1024).
void part_range(const scape* h, int i, int n, int64_t* first, int64_t* end) {
  const int64_t tiles_all = (h->n_chunks + 7) / 8;
  *first = 1024 * (tiles_all * i / n);
  *end = i + 1 == n ? h->N : std::min<int64_t>(h->N, 1024 * (tiles_all * (i + 1) / n));
}

// scape_step_host's pipeline: the streaming kernel runs part by part, `before(i, n)` / `after(i, n)` around
// each launch (upload / download of that part); n = 1 when the step cannot be split (all-ones mask, dense m,
// layers, clip_grad, a shard of too few tiles).
struct PartHooks {
  int n_parts;
  std::function<int(int, int)> before, after;
};

// The step.  local = false: all of it (scape_step).  local = true (scape_step_local): everything
// that needs no other worker -- l.6-9 for the local replicas, the local sums of l.10 parked for the
// all-reduce, theta off the mask, this worker's share of the refresh (l.11) -- and the rest is left
// to scape_step_apply.
int step_impl(scape_t* h, float* param, const void* const* grads, void* cuda_stream, bool local, const PartHooks* hooks = nullptr) {
  if (!h) return fail(SCAPE_EINVAL, "NULL handle");
  if (h->pending) return fail(SCAPE_EINVAL, "scape_step_local has run: call scape_step_apply first");
  if (!local && h->world > 1) return fail(SCAPE_EINVAL, "this handle is one of %d workers: use scape_step_local / scape_step_apply", h->world);
  if (local && h->clip_max_norm > 0.0) return fail(SCAPE_EINVAL, "clip_grad is not available with scape_step_local");
  if (local && !h->ghat) return fail(SCAPE_EINVAL, "call scape_set_workers before scape_step_local");
  if (!param || !grads) return fail(SCAPE_EINVAL, "NULL param/grads");
  if ((uintptr_t)param & 15) return fail(SCAPE_EINVAL, "param must be 16-byte aligned");
  for (int r = 0; r < h->R; ++r) {
    if (!grads[r]) return fail(SCAPE_EINVAL, "grads[%d] is NULL", r);
    if ((uintptr_t)grads[r] & 15) return fail(SCAPE_EINVAL, "grads[%d] must be 16-byte aligned", r);
  }
  DeviceGuard guard(h->dev);
  if (!guard.ok) return fail(SCAPE_ECUDA, "cannot select the handle's device");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int rc;
  if ((rc = join_side(h, st))) return rc;      // M_{t-1} (rank, index list, predicted bracket) may still be on its way

  MaskSlot& cur = h->slot[h->use];
  MaskSlot& nxt = h->slot[h->build];
  const bool need_select = h->k < h->N;
  // stage 2 on the handle's own stream, off the caller's: never inside a capture
  const bool async = h->async_refresh && need_select && !local && !is_capturing(st);
  // an all-ones step reads and writes m densely
  if (cur.all_ones && h->m_sparse) {
    if ((rc = materialise_dense_m(h, st))) return rc;
    h->m_sparse = false;
  }
  const bool msparse = h->m_sparse;
  const int pm_out = msparse ? 1 - h->pm_last : 0;

  StepParams p{};
  p.theta = param; p.m = h->m; p.e = h->e; p.e_stride = h->Npad;
  for (int r = 0; r < h->R; ++r) p.g[r] = grads[r];
  p.cur_bits = cur.bits; p.cur_rk = cur.rank; p.cur_pre = cur.pre; p.cur_trank = cur.trank;
  p.packed = cur.all_ones ? h->dense_pack : h->packed;
  p.packed_stride = cur.all_ones ? h->Npad : h->packed_stride;
  p.packed_mean = h->pm[pm_out];
  if (msparse) {
    p.prev_bits = h->slot[h->last].bits; p.prev_rk = h->slot[h->last].rank; p.prev_pre = h->slot[h->last].pre; p.prev_trank = h->slot[h->last].trank; p.pm_prev = h->pm[h->pm_last];
  }
  p.N = h->N; p.n_chunks = h->n_chunks;
  p.b1 = h->b1; p.c1 = h->c1; p.b2 = h->b2; p.c2 = h->c2; p.eps = h->eps; p.wd = h->wd; p.neg_lr = -h->lr;
  p.R_f = (float)h->R; p.inv_R = 1.0f / (float)h->R;
  p.r_pow2 = (h->R & (h->R - 1)) == 0;      // x / 2^n == x * 2^-n bit for bit
  p.stash = cur.all_ones && need_select;
  p.bc1 = 1.0f; p.bc2 = 1.0f;
  if (h->bias_correction) {      // PAPER.md:77; factors evaluated in double from the step number, cast once
    const double t = (double)(h->t + 1);
    p.bc1 = (float)(1.0 / (1.0 - std::pow(h->beta1_d, t)));
    p.bc2 = (float)(1.0 / (1.0 - std::pow(h->beta2_d, t)));
  }
  const bool clip = !local && h->clip_max_norm > 0.0;
  p.clip = local ? 2 : clip ? 1 : 0; p.ghat = h->ghat; p.vm = h->vm; p.sumsq = h->sumsq;
  p.ctl = h->sel; p.next_bits = nxt.bits; p.cand = h->cand;
  p.seg_count = h->seg_count; p.seg_above = h->seg_above;
  if (h->n_layers > 0) { p.chunk_layer = h->chunk_layer; p.layers = h->layers; }

  const bool prof = h->prof_on;
  if (prof && h->prof_pending == scape::kProfRing) { int prc = prof_drain(h); if (prc) return prc; }
  const int pi = h->prof_pending;
  if (prof) CU_TRY(cudaEventRecord(h->prof_ev[pi][0], st));
  if (hooks) {
    int n = hooks->n_parts;
    if (cur.all_ones || !msparse || h->n_layers > 0 || p.clip || p.N / kTmaTile < (int64_t)h->n_sm * 2 * n) n = 1;
    if (n > 1) {                 // parts with fewer CTAs than the full grid leave segments untouched: their counts must read 0
      CU_TRY(cudaMemsetAsync(h->seg_count, 0, sizeof(uint32_t) * h->max_seg, st));
      CU_TRY(cudaMemsetAsync(h->seg_above, 0, sizeof(uint32_t) * h->max_seg, st));
    }
    for (int i = 0; i < n; ++i) {
      if ((rc = hooks->before(i, n))) return rc;
      if ((rc = launch_fused(h, p, cur.all_ones, msparse, st, i, n))) return rc;
      if ((rc = hooks->after(i, n))) return rc;
    }
  } else {
    rc = launch_fused(h, p, cur.all_ones, msparse, st);
    if (rc) return rc;
  }
  if (clip) {
    // l.14-17 on the mask: norm of g^ (fixed-order reduction), then the deferred update
    const int64_t K = cur.count;
    clip_norm_kernel<<<1, 1024, 0, st>>>(h->sumsq, h->n_slots, h->clip_max_norm, h->clip_state);
    int g2 = (int)((K + 255) / 256); if (g2 > h->n_sm * 16) g2 = h->n_sm * 16; if (g2 < 1) g2 = 1;
    clip_update_kernel<<<g2, 256, 0, st>>>(param, cur.all_ones ? nullptr : cur.idx, cur.all_ones ? h->m : h->pm[pm_out],
                                           h->ghat, h->vm, K, h->clip_state, h->c2, h->eps, h->wd, -h->lr, p.bc1, p.bc2);
    h->launches += 2;
    CU_TRY(cudaGetLastError());
  }
  if (prof) CU_TRY(cudaEventRecord(h->prof_ev[pi][1], st));

  cudaStream_t ss = st;                        // the stream stage 2 runs on
  if (async) { if ((rc = fork_side(h, st))) return rc; ss = h->side; }
  if (need_select) {
    // workers: an all-ones step does not write M_t in the fused pass, and the select only writes
    // this worker's layers: the others' words must read zero for the exchange
    if (local && cur.all_ones && h->n_layers > 0) CU_TRY(cudaMemsetAsync(nxt.bits, 0, sizeof(uint32_t) * h->n_words, ss));
    rc = h->n_layers > 0 ? run_select_layered(h, cur, nxt, /*force_general=*/cur.all_ones, ss, /*compact=*/!local)
                         : run_select(h, cur, nxt, /*force_general=*/cur.all_ones, ss, /*compact=*/!local);
    if (rc) return rc;
    if (cur.all_ones) CU_TRY(cudaMemsetAsync(h->e, 0, sizeof(float) * h->Npad, ss));   // l.8 for e^0 after the stash
  } else if (!local) {
    nxt.all_ones = true; nxt.count = h->N; nxt.valid = true;                            // k = N: M_t = 1
  }
  if (prof) { CU_TRY(cudaEventRecord(h->prof_ev[pi][2], ss)); h->prof_pending = pi + 1; }
  if (async && (rc = mark_side(h))) return rc;
  if (local) {
    h->pending = true; h->pending_pm_out = pm_out; h->pending_bc1 = p.bc1; h->pending_bc2 = p.bc2; h->pending_lr = h->lr;
    h->pending_need_select = need_select;
    return SCAPE_OK;
  }
  h->last_dense = cur.all_ones;
  if (!cur.all_ones) { h->m_sparse = true; h->pm_last = pm_out; }   // m_t = b-_t, addressed through `cur`
  { const int old_last = h->last; h->last = h->use; h->use = h->build; h->build = old_last; }
  h->lr_last = h->lr;
  h->t += 1;
  return SCAPE_OK;
}

}  // namespace

extern "C" int scape_step(scape_t* h, float* param, const void* const* grads, void* cuda_stream) {
  return step_impl(h, param, grads, cuda_stream, /*local=*/false);
}

// ---- workers: PAPER.md:136 (N workers), :155 (all-reduce of b), :178 / :218 (each worker refreshes
// ---- a portion of the mask, the portions are gathered)  --  SURVEY.md §8(f) rank 3
extern "C" int scape_set_workers(scape_t* h, int world, int rank, const int32_t* layer_owner) {
  if (!h) return fail(SCAPE_EINVAL, "NULL handle");
  if (world < 1 || rank < 0 || rank >= world) return fail(SCAPE_EINVAL, "need 0 <= rank < world");
  if (h->pending) return fail(SCAPE_EINVAL, "a split step is in flight");
  if (world > 1 && (h->n_layers == 0 || !layer_owner))
    return fail(SCAPE_EINVAL, "more than one worker needs layers (scape_set_layers) and an owner per layer");
  if (layer_owner && h->n_layers == 0) return fail(SCAPE_EINVAL, "layer owners need layers (scape_set_layers)");
  if (layer_owner)
    for (int l = 0; l < h->n_layers; ++l)
      if (layer_owner[l] < 0 || layer_owner[l] >= world) return fail(SCAPE_EINVAL, "layer_owner[%d] out of range", l);
  DeviceGuard g(h->dev);
  CU_TRY(cudaDeviceSynchronize());
  if (!h->ghat) {                      // exchange buffers: the local sums and m_old of the selected entries
    if (cudaMalloc((void**)&h->ghat, sizeof(float) * h->Npad) != cudaSuccess ||
        cudaMalloc((void**)&h->vm, sizeof(float) * h->Npad) != cudaSuccess) {
      cudaGetLastError();
      cudaFree(h->ghat); cudaFree(h->vm); h->ghat = h->vm = nullptr;
      return fail(SCAPE_ENOMEM, "set_workers: allocation of 2 N floats failed");
    }
  }
  if (h->n_layers > 0) {
    std::vector<LayerState> ls((size_t)h->n_layers);
    CU_TRY(cudaMemcpy(ls.data(), h->layers, sizeof(LayerState) * ls.size(), cudaMemcpyDeviceToHost));
    h->lay_skip.assign((size_t)h->n_layers, 0);
    for (int l = 0; l < h->n_layers; ++l) {
      LayerState& S = ls[(size_t)l];
      const int skip = layer_owner ? (layer_owner[l] != rank) : 0;
      if (skip != S.skip) {            // ownership changed: forget the prediction
        S.skip = skip;
        S.br = Bracket{};
        S.br.delta = 0.5f;
        S.br.lo_key = S.br.hi_key = (skip || S.compress) ? 0xFFFFFFFFu : 0u;
      }
      h->lay_skip[(size_t)l] = (uint8_t)skip;
    }
    CU_TRY(cudaMemcpy(h->layers, ls.data(), sizeof(LayerState) * ls.size(), cudaMemcpyHostToDevice));
  }
  h->world = world; h->rank = rank;
  build_exchange_plan(h, world > 1 ? layer_owner : nullptr);
  cudaFree(h->x_shared_idx); cudaFree(h->x_shared_buf);
  h->x_shared_idx = h->x_shared_buf = nullptr;
  if (!h->x_shared.empty()) {
    std::vector<uint32_t> w(h->x_shared.begin(), h->x_shared.end());
    if (cudaMalloc((void**)&h->x_shared_idx, sizeof(uint32_t) * w.size()) != cudaSuccess ||
        cudaMalloc((void**)&h->x_shared_buf, sizeof(uint32_t) * w.size()) != cudaSuccess) {
      cudaGetLastError();
      return fail(SCAPE_ENOMEM, "set_workers: allocation of the shared-word list failed");
    }
    CU_TRY(cudaMemcpy(h->x_shared_idx, w.data(), sizeof(uint32_t) * w.size(), cudaMemcpyHostToDevice));
  }
  return SCAPE_OK;
}

extern "C" int scape_step_local(scape_t* h, float* param, const void* const* grads, void* cuda_stream) {
  return step_impl(h, param, grads, cuda_stream, /*local=*/true);
}

extern "C" int scape_exchange_buffers(scape_t* h, float** sums, int64_t* n_sums, uint32_t** mask_words, int64_t* n_mask_words) {
  if (!h) return fail(SCAPE_EINVAL, "NULL handle");
  if (!h->pending) return fail(SCAPE_EINVAL, "no split step is in flight (call scape_step_local first)");
  const MaskSlot& cur = h->slot[h->use];
  if (sums) *sums = h->ghat;
  if (n_sums) *n_sums = cur.all_ones ? h->N : cur.count;
  if (mask_words) *mask_words = h->pending_need_select ? h->slot[h->build].bits : nullptr;
  if (n_mask_words) *n_mask_words = h->pending_need_select ? h->n_words : 0;
  return SCAPE_OK;
}

extern "C" int scape_step_apply(scape_t* h, float* param, void* cuda_stream) {
  if (!h) return fail(SCAPE_EINVAL, "NULL handle");
  if (!param) return fail(SCAPE_EINVAL, "NULL param");
  if (!h->pending) return fail(SCAPE_EINVAL, "no split step is in flight (call scape_step_local first)");
  DeviceGuard guard(h->dev);
  if (!guard.ok) return fail(SCAPE_ECUDA, "cannot select the handle's device");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  MaskSlot& cur = h->slot[h->use];
  MaskSlot& nxt = h->slot[h->build];
  const int pm_out = h->pending_pm_out;
  if (h->pending_need_select && is_capturing(st) && h->pending_mask_on_side)
    return fail(SCAPE_EINVAL, "a mask exchange on the handle's own stream cannot be part of a captured graph");
  const int64_t K = cur.all_ones ? h->N : cur.count;
  const int Rt = h->R * h->world;
  int g2 = (int)((K + 255) / 256); if (g2 > h->n_sm * 16) g2 = h->n_sm * 16; if (g2 < 1) g2 = 1;
  dist_update_kernel<<<g2, 256, 0, st>>>(param, cur.all_ones ? nullptr : cur.idx, cur.all_ones ? h->m : h->pm[pm_out],
                                         h->ghat, h->vm, K, (float)Rt, 1.0f / (float)Rt, (Rt & (Rt - 1)) == 0 ? 1 : 0,
                                         h->b1, h->c1, h->b2, h->c2, h->eps, h->wd, -h->pending_lr, h->pending_bc1, h->pending_bc2);
  h->launches++;
  CU_TRY(cudaGetLastError());
  if (h->pending_need_select) {
    // M_t is complete now: rank128 + the index list -- on the handle's own stream when the mask
    // portions travelled there (scape_step_exchange with a mask_comm); the next step waits for it
    cudaStream_t cs = h->pending_mask_on_side ? h->side : st;
    int rc = compact_mask(h, nxt, true, cs);
    if (rc) return rc;
    if (h->pending_mask_on_side) { if ((rc = mark_side(h))) return rc; h->pending_mask_on_side = false; }
    nxt.count = h->k; nxt.all_ones = false; nxt.valid = true;
  } else {
    nxt.all_ones = true; nxt.count = h->N; nxt.valid = true;
  }
  h->pending = false;
  h->last_dense = cur.all_ones;
  if (!cur.all_ones) { h->m_sparse = true; h->pm_last = pm_out; }
  { const int old_last = h->last; h->last = h->use; h->use = h->build; h->build = old_last; }
  h->lr_last = h->pending_lr;
  h->t += 1;
  return SCAPE_OK;
}

// ---- the exchange inside the library ---------------------
extern "C" int scape_step_exchange(scape_t* h, void* comm, void* mask_comm, void* cuda_stream) {
  if (!h) return fail(SCAPE_EINVAL, "NULL handle");
  if (!h->pending) return fail(SCAPE_EINVAL, "no split step is in flight (call scape_step_local first)");
  if (!comm) return fail(SCAPE_EINVAL, "NULL communicator");
  if (h->pending_mask_on_side) return fail(SCAPE_EINVAL, "this split step has been exchanged already");
  const NcclApi* nc = nccl();
  if (!nc) return fail(SCAPE_ECUDA, "NCCL (libnccl.so.2) could not be loaded: %s", dlerror() ? dlerror() : "symbol missing");
  DeviceGuard guard(h->dev);
  if (!guard.ok) return fail(SCAPE_ECUDA, "cannot select the handle's device");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const MaskSlot& cur = h->slot[h->use];
  const int64_t n_sums = cur.all_ones ? h->N : cur.count;
  // l.10: the local sums of every selected entry become the sum over all workers
  if (n_sums > 0) NCCL_TRY(nc, nc->AllReduce(h->ghat, h->ghat, (size_t)n_sums, kNcclFloat32, kNcclSum, comm, st));
  if (!h->pending_need_select) return SCAPE_OK;
  // M_t: only what each worker made travels, from its owner; on the handle's own stream when it has
  // a communicator of its own (the one-step delay: nobody needs M_t before the next step's local half)
  const bool on_side = mask_comm != nullptr && mask_comm != comm && !is_capturing(st);
  cudaStream_t ms = st;
  void* mc = mask_comm ? mask_comm : comm;
  if (on_side) { int rc = fork_side(h, st); if (rc) return rc; ms = h->side; }
  uint32_t* bits = h->slot[h->build].bits;
  NCCL_TRY(nc, nc->GroupStart());
  for (size_t i = 0; i < h->xr_first.size(); ++i) {
    int r = nc->Broadcast(bits + h->xr_first[i], bits + h->xr_first[i], (size_t)(h->xr_end[i] - h->xr_first[i]), kNcclUint32,
                          h->xr_owner[i], mc, ms);
    if (r != 0) { nc->GroupEnd(); return fail(SCAPE_ECUDA, "ncclBroadcast: %s", nc->GetErrorString(r)); }
  }
  NCCL_TRY(nc, nc->GroupEnd());
  const int ns = (int)h->x_shared.size();
  if (ns > 0) {
    gather_words_kernel<<<(ns + 255) / 256, 256, 0, ms>>>(bits, h->x_shared_idx, ns, h->x_shared_buf);
    NCCL_TRY(nc, nc->AllReduce(h->x_shared_buf, h->x_shared_buf, (size_t)ns, kNcclUint32, kNcclSum, mc, ms));   // disjoint bits: SUM = OR
    scatter_words_kernel<<<(ns + 255) / 256, 256, 0, ms>>>(bits, h->x_shared_idx, ns, h->x_shared_buf);
    h->launches += 2;
    CU_TRY(cudaGetLastError());
  }
  h->pending_mask_on_side = on_side;
  return SCAPE_OK;
}

extern "C" int scape_exchange_plan(const scape_t* h, int64_t* first, int64_t* end, int32_t* owner, int cap, int* n_ranges,
                                   int64_t* shared, int cap_shared, int* n_shared) {
  if (!h) return fail(SCAPE_EINVAL, "NULL handle");
  const int nr = (int)h->xr_first.size(), ns = (int)h->x_shared.size();
  if (n_ranges) *n_ranges = nr;
  if (n_shared) *n_shared = ns;
  if ((first || end || owner) && cap < nr) return fail(SCAPE_EINVAL, "exchange_plan: %d ranges, capacity %d", nr, cap);
  if (shared && cap_shared < ns) return fail(SCAPE_EINVAL, "exchange_plan: %d shared words, capacity %d", ns, cap_shared);
  for (int i = 0; i < nr; ++i) {
    if (first) first[i] = h->xr_first[i];
    if (end) end[i] = h->xr_end[i];
    if (owner) owner[i] = h->xr_owner[i];
  }
  for (int i = 0; i < ns && shared; ++i) shared[i] = h->x_shared[i];
  return SCAPE_OK;
}

extern "C" int scape_nccl_unique_id(void* id) {
  if (!id) return fail(SCAPE_EINVAL, "NULL id");
  const NcclApi* nc = nccl();
  if (!nc) return fail(SCAPE_ECUDA, "NCCL (libnccl.so.2) could not be loaded");
  NCCL_TRY(nc, nc->GetUniqueId((NcclId*)id));
  return SCAPE_OK;
}

extern "C" int scape_nccl_comm_create(int world, int rank, const void* id, void** comm) {
  if (!id || !comm || world < 1 || rank < 0 || rank >= world) return fail(SCAPE_EINVAL, "bad argument");
  const NcclApi* nc = nccl();
  if (!nc) return fail(SCAPE_ECUDA, "NCCL (libnccl.so.2) could not be loaded");
  NcclId uid;
  std::memcpy(&uid, id, sizeof uid);
  NCCL_TRY(nc, nc->CommInitRank(comm, world, uid, rank));
  return SCAPE_OK;
}

extern "C" int scape_nccl_comm_destroy(void* comm) {
  if (!comm) return SCAPE_OK;
  const NcclApi* nc = nccl();
  if (!nc) return fail(SCAPE_ECUDA, "NCCL (libnccl.so.2) could not be loaded");
  NCCL_TRY(nc, nc->CommDestroy(comm));
  return SCAPE_OK;
}

// ---- asynchronous refresh ------------------------------------------------
extern "C" int scape_set_async_refresh(scape_t* h, int on) {
  if (!h) return fail(SCAPE_EINVAL, "NULL handle");
  if (h->pending) return fail(SCAPE_EINVAL, "a split step is in flight");
  DeviceGuard g(h->dev);
  if (on) { int rc = ensure_side(h); if (rc) return rc; }
  h->async_refresh = on != 0;
  return SCAPE_OK;
}

extern "C" int scape_join_refresh(scape_t* h, void* cuda_stream) {
  if (!h) return fail(SCAPE_EINVAL, "NULL handle");
  DeviceGuard g(h->dev);
  return join_side(h, (cudaStream_t)cuda_stream);
}

// ---- Algorithm 2, parameter side (Eq. 6 :207-211)  --  SURVEY.md §8(f) rank 4
extern "C" int scape_param_pack(scape_t* h, const float* param, int64_t first, int64_t count, void* out, int dtype,
                                void* cuda_stream) {
  if (!h) return fail(SCAPE_EINVAL, "NULL handle");
  if (h->pending) return fail(SCAPE_EINVAL, "a split step is in flight: scape_step_apply first");
  if (dtype != SCAPE_PARAM_F32 && dtype != SCAPE_PARAM_BF16) return fail(SCAPE_EINVAL, "unknown payload dtype %d", dtype);
  const MaskSlot& la = h->slot[h->last];
  if (h->t == 0 || !la.valid) return fail(SCAPE_EINVAL, "no step has run yet: there is no updated parameter to send");
  if (first < 0 || count < 0 || first + count > la.count)
    return fail(SCAPE_EINVAL, "range [%lld, %lld) outside the %lld entries of the mask the last step used", (long long)first,
                (long long)(first + count), (long long)la.count);
  if (count == 0) return SCAPE_OK;
  if (!param || !out) return fail(SCAPE_EINVAL, "NULL param/out");
  if ((uintptr_t)out & (dtype == SCAPE_PARAM_BF16 ? 1 : 3)) return fail(SCAPE_EINVAL, "out is misaligned for its element type");
  DeviceGuard guard(h->dev);
  if (!guard.ok) return fail(SCAPE_ECUDA, "cannot select the handle's device");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  { const int jr = join_side(h, st); if (jr) return jr; }     // a refresh on the handle's own stream comes first
  int64_t grid = (count + 1023) / 1024; if (grid > h->n_sm * 16) grid = h->n_sm * 16;
  const int32_t* idx = la.all_ones ? nullptr : la.idx;
  if (dtype == SCAPE_PARAM_BF16) param_pack_kernel<true><<<(int)grid, 256, 0, st>>>(param, idx, first, count, out);
  else param_pack_kernel<false><<<(int)grid, 256, 0, st>>>(param, idx, first, count, out);
  h->launches++;
  CU_TRY(cudaGetLastError());
  return SCAPE_OK;
}

extern "C" int scape_param_apply(scape_t* h, float* w, void* w_hat, const void* payload, int dtype, void* cuda_stream) {
  if (!h) return fail(SCAPE_EINVAL, "NULL handle");
  if (h->pending) return fail(SCAPE_EINVAL, "a split step is in flight: scape_step_apply first");
  if (dtype != SCAPE_PARAM_F32 && dtype != SCAPE_PARAM_BF16) return fail(SCAPE_EINVAL, "unknown payload dtype %d", dtype);
  MaskSlot& la = h->slot[h->last];
  if (h->t == 0 || !la.valid) return fail(SCAPE_EINVAL, "no step has run yet");
  if (!w || (!payload && la.count > 0)) return fail(SCAPE_EINVAL, "NULL w/payload");
  if ((uintptr_t)w & 15) return fail(SCAPE_EINVAL, "w must be 16-byte aligned");
  if ((uintptr_t)w_hat & 7) return fail(SCAPE_EINVAL, "w_hat must be 8-byte aligned");
  if ((uintptr_t)payload & (dtype == SCAPE_PARAM_BF16 ? 1 : 3)) return fail(SCAPE_EINVAL, "payload is misaligned for its element type");
  DeviceGuard guard(h->dev);
  if (!guard.ok) return fail(SCAPE_ECUDA, "cannot select the handle's device");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  { const int jr = join_side(h, st); if (jr) return jr; }     // a refresh on the handle's own stream comes first
  const int grid = grid_for(h, (h->n_chunks + kApplyChunks - 1) / kApplyChunks, 8, 4);
  const bool bf = dtype == SCAPE_PARAM_BF16, hat = w_hat != nullptr, ones = la.all_ones;
  const float wd = h->wd, neg_lr = -h->lr_last;
  uint16_t* wh = (uint16_t*)w_hat;
#define SCAPE_APPLY(B_, H_, O_) param_apply_kernel<B_, H_, O_><<<grid, 256, 0, st>>>(w, wh, la.bits, la.rank, payload, h->N, h->n_chunks, wd, neg_lr)
  if (ones) { if (bf) { if (hat) SCAPE_APPLY(true, true, true); else SCAPE_APPLY(true, false, true); }
              else    { if (hat) SCAPE_APPLY(false, true, true); else SCAPE_APPLY(false, false, true); } }
  else      { if (bf) { if (hat) SCAPE_APPLY(true, true, false); else SCAPE_APPLY(true, false, false); }
              else    { if (hat) SCAPE_APPLY(false, true, false); else SCAPE_APPLY(false, false, false); } }
#undef SCAPE_APPLY
  h->launches++;
  CU_TRY(cudaGetLastError());
  return SCAPE_OK;
}

// ---- mask bit pack / unpack, stand-alone: no handle ----------------------
extern "C" int scape_mask_pack(const uint8_t* mask_bytes, int64_t n, uint32_t* words, void* cuda_stream) {
  if (n < 0) return fail(SCAPE_EINVAL, "n must be >= 0");
  if (n == 0) return SCAPE_OK;
  if (!mask_bytes || !words) return fail(SCAPE_EINVAL, "NULL argument");
  if ((uintptr_t)words & 3) return fail(SCAPE_EINVAL, "words must be 4-byte aligned");
  const int64_t groups = (n + 31) >> 5;
  int64_t grid = (groups + 255) / 256; if (grid > 148 * 32) grid = 148 * 32;
  mask_pack_kernel<<<(int)grid, 256, 0, (cudaStream_t)cuda_stream>>>(mask_bytes, n, words);
  CU_TRY(cudaGetLastError());
  return SCAPE_OK;
}

extern "C" int scape_mask_unpack(const uint32_t* words, int64_t n, uint8_t* mask_bytes, void* cuda_stream) {
  if (n < 0) return fail(SCAPE_EINVAL, "n must be >= 0");
  if (n == 0) return SCAPE_OK;
  if (!mask_bytes || !words) return fail(SCAPE_EINVAL, "NULL argument");
  if ((uintptr_t)words & 3) return fail(SCAPE_EINVAL, "words must be 4-byte aligned");
  const int64_t groups = (n + 15) >> 4;
  int64_t grid = (groups + 255) / 256; if (grid > 148 * 32) grid = 148 * 32;
  mask_unpack_kernel<<<(int)grid, 256, 0, (cudaStream_t)cuda_stream>>>(words, n, mask_bytes);
  CU_TRY(cudaGetLastError());
  return SCAPE_OK;
}

extern "C" int scape_select_stats(scape_t* h, int64_t* fast, int64_t* general, void* cuda_stream) {
  if (!h) return fail(SCAPE_EINVAL, "NULL handle");
  DeviceGuard guard(h->dev);
  { const int jr = join_side(h, (cudaStream_t)cuda_stream); if (jr) return jr; }     // a refresh on the handle's own stream comes first
  SelState s{};
  LayerCtl lc{};
  CU_TRY(cudaMemcpyAsync(&s, h->sel, sizeof s, cudaMemcpyDeviceToHost, (cudaStream_t)cuda_stream));
  if (h->lctl) CU_TRY(cudaMemcpyAsync(&lc, h->lctl, sizeof lc, cudaMemcpyDeviceToHost, (cudaStream_t)cuda_stream));
  CU_TRY(cudaStreamSynchronize((cudaStream_t)cuda_stream));
  if (fast) *fast = (int64_t)(s.n_fast + lc.n_fast);
  if (general) *general = (int64_t)(s.n_general + lc.n_general);
  return SCAPE_OK;
}

extern "C" int scape_select_recovered(scape_t* h, int64_t* recovered, void* cuda_stream) {
  if (!h || !recovered) return fail(SCAPE_EINVAL, "NULL argument");
  DeviceGuard guard(h->dev);
  { const int jr = join_side(h, (cudaStream_t)cuda_stream); if (jr) return jr; }
  SelState s{};
  CU_TRY(cudaMemcpyAsync(&s, h->sel, sizeof s, cudaMemcpyDeviceToHost, (cudaStream_t)cuda_stream));
  CU_TRY(cudaStreamSynchronize((cudaStream_t)cuda_stream));
  *recovered = (int64_t)s.n_recovered;
  return SCAPE_OK;
}

extern "C" int scape_select_debug(scape_t* h, double* out8, void* cuda_stream) {
  if (!h || !out8) return fail(SCAPE_EINVAL, "NULL argument");
  DeviceGuard guard(h->dev);
  { const int jr = join_side(h, (cudaStream_t)cuda_stream); if (jr) return jr; }     // a refresh on the handle's own stream comes first
  SelState s{};
  CU_TRY(cudaMemcpyAsync(&s, h->sel, sizeof s, cudaMemcpyDeviceToHost, (cudaStream_t)cuda_stream));
  CU_TRY(cudaStreamSynchronize((cudaStream_t)cuda_stream));
  out8[0] = s.hit; out8[1] = (double)s.n_above; out8[2] = (double)s.n_cand; out8[3] = s.br.delta;
  out8[4] = s.br.lnT_prev; out8[5] = s.br.ln_pred; out8[6] = (double)s.cand_cap_total; out8[7] = (double)h->n_seg;
  return SCAPE_OK;
}

extern "C" int scape_profile(scape_t* h, int on) {
  if (!h) return fail(SCAPE_EINVAL, "NULL handle");
  DeviceGuard guard(h->dev);
  if (on && !h->prof_have_events) {
    for (auto& row : h->prof_ev) for (auto& ev : row) CU_TRY(cudaEventCreate(&ev));
    h->prof_have_events = true;
  }
  if (h->prof_on) { int rc = prof_drain(h); if (rc) return rc; }
  h->prof_on = on != 0;
  h->prof_fused_ms = h->prof_select_ms = 0.0;
  h->prof_steps = 0;
  return SCAPE_OK;
}

extern "C" int scape_profile_read(scape_t* h, double* fused_ms, double* select_ms, int64_t* steps) {
  if (!h) return fail(SCAPE_EINVAL, "NULL handle");
  DeviceGuard guard(h->dev);
  int rc = prof_drain(h);
  if (rc) return rc;
  if (fused_ms) *fused_ms = h->prof_fused_ms;
  if (select_ms) *select_ms = h->prof_select_ms;
  if (steps) *steps = h->prof_steps;
  return SCAPE_OK;
}

extern "C" int scape_step_host(scape_t* h, float* param_host, const void* const* grads_host, void* cuda_stream) {
  if (!h) return fail(SCAPE_EINVAL, "NULL handle");
  if (!param_host || !grads_host) return fail(SCAPE_EINVAL, "NULL param/grads");
  DeviceGuard guard(h->dev);
  if (!guard.ok) return fail(SCAPE_ECUDA, "cannot select the handle's device");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const size_t gb = (size_t)h->N * (h->grad_dtype == SCAPE_GRAD_BF16 ? 2 : 4);
  if (!h->st_param) {
    if (cudaMalloc((void**)&h->st_param, sizeof(float) * h->N) != cudaSuccess) { h->st_param = nullptr; cudaGetLastError(); return fail(SCAPE_ENOMEM, "staging allocation failed"); }
  }
  if (h->st_grad_bytes != gb) {
    for (int r = 0; r < h->R; ++r) {
      cudaFree(h->st_grad[r]); h->st_grad[r] = nullptr;
      if (cudaMalloc(&h->st_grad[r], gb) != cudaSuccess) { h->st_grad[r] = nullptr; h->st_grad_bytes = 0; cudaGetLastError(); return fail(SCAPE_ENOMEM, "staging allocation failed"); }
    }
    h->st_grad_bytes = gb;
  }
  for (int r = 0; r < h->R; ++r)
    if (!grads_host[r]) return fail(SCAPE_EINVAL, "grads[%d] is NULL", r);
  // Upload, step and download are pipelined part by part: PCIe is full duplex and the streaming kernel is
  // 2.5 % of the copies' time, so theta of part i travels back while the gradients of part i + 1 travel up.
  // Two streams of the handle's own carry the copies; events order them against the kernel launches on st.
  if (!h->up) {
    CU_TRY(cudaStreamCreateWithFlags(&h->up, cudaStreamNonBlocking));
    CU_TRY(cudaStreamCreateWithFlags(&h->down, cudaStreamNonBlocking));
    for (auto& e : h->ev_up) CU_TRY(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    for (auto& e : h->ev_cmp) CU_TRY(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    CU_TRY(cudaEventCreateWithFlags(&h->ev_host, cudaEventDisableTiming));
  }
  const size_t ge = h->grad_dtype == SCAPE_GRAD_BF16 ? 2 : 4;
  CU_TRY(cudaEventRecord(h->ev_host, st));                       // the copies come after whatever st already holds
  CU_TRY(cudaStreamWaitEvent(h->up, h->ev_host, 0));
  CU_TRY(cudaStreamWaitEvent(h->down, h->ev_host, 0));
  PartHooks hooks;
  hooks.n_parts = scape::kHostParts;
  hooks.before = [&](int i, int n) -> int {
    int64_t a, b;
    part_range(h, i, n, &a, &b);
    for (int r = 0; r < h->R; ++r)
      CU_TRY(cudaMemcpyAsync((char*)h->st_grad[r] + a * ge, (const char*)grads_host[r] + a * ge, (size_t)(b - a) * ge, cudaMemcpyHostToDevice, h->up));
    CU_TRY(cudaMemcpyAsync(h->st_param + a, param_host + a, sizeof(float) * (size_t)(b - a), cudaMemcpyHostToDevice, h->up));
    CU_TRY(cudaEventRecord(h->ev_up[i], h->up));
    CU_TRY(cudaStreamWaitEvent(st, h->ev_up[i], 0));
    return SCAPE_OK;
  };
  hooks.after = [&](int i, int n) -> int {
    int64_t a, b;
    part_range(h, i, n, &a, &b);
    CU_TRY(cudaEventRecord(h->ev_cmp[i], st));
    CU_TRY(cudaStreamWaitEvent(h->down, h->ev_cmp[i], 0));
    if (h->clip_max_norm > 0.0 && n == 1) return SCAPE_OK;       // clip_grad finishes theta after the kernel: copied below
    CU_TRY(cudaMemcpyAsync(param_host + a, h->st_param + a, sizeof(float) * (size_t)(b - a), cudaMemcpyDeviceToHost, h->down));
    return SCAPE_OK;
  };
  int rc = step_impl(h, h->st_param, (const void* const*)h->st_grad, cuda_stream, /*local=*/false, &hooks);
  if (rc) return rc;
  if (h->clip_max_norm > 0.0) CU_TRY(cudaMemcpyAsync(param_host, h->st_param, sizeof(float) * h->N, cudaMemcpyDeviceToHost, st));
  CU_TRY(cudaEventRecord(h->ev_host, h->down));
  CU_TRY(cudaStreamWaitEvent(st, h->ev_host, 0));
  CU_TRY(cudaStreamSynchronize(st));
  return SCAPE_OK;
}

// ---------------------------------------------------------------------------------------------
// accessors
// ---------------------------------------------------------------------------------------------
namespace {

int materialise_all_ones(scape* h, MaskSlot& s, cudaStream_t st) {
  mask_all_ones_kernel<<<256, 256, 0, st>>>(s.bits, h->n_words, h->N);
  h->launches++;
  CU_TRY(cudaGetLastError());
  return SCAPE_OK;
}

int get_idx(scape* h, MaskSlot& s, void* buf, size_t bytes, cudaStream_t st) {
  if (bytes != sizeof(int32_t) * (size_t)s.count) return fail(SCAPE_EINVAL, "idx: expected %zu bytes", sizeof(int32_t) * (size_t)s.count);
  if (!s.all_ones) {
    CU_TRY(cudaMemcpyAsync(buf, s.idx, bytes, cudaMemcpyDefault, st));
    return SCAPE_OK;
  }
  // all-ones mask: the list is 0 .. N-1, produced piecewise in a small scratch kept by the handle
  constexpr int64_t kPiece = 1 << 20;
  if (!h->iota_scratch) {
    if (cudaMalloc((void**)&h->iota_scratch, sizeof(int32_t) * kPiece) != cudaSuccess) {
      h->iota_scratch = nullptr; cudaGetLastError();
      return fail(SCAPE_ENOMEM, "idx: scratch allocation failed");
    }
  }
  for (int64_t lo = 0; lo < h->N; lo += kPiece) {
    const int64_t n = std::min<int64_t>(kPiece, h->N - lo);
    iota_i32_kernel<<<256, 256, 0, st>>>(h->iota_scratch, n, (int32_t)lo);
    h->launches++;
    CU_TRY(cudaMemcpyAsync((char*)buf + sizeof(int32_t) * (size_t)lo, h->iota_scratch, sizeof(int32_t) * (size_t)n, cudaMemcpyDefault, st));
    CU_TRY(cudaStreamSynchronize(st));        // the scratch is reused by the next piece (the copy may be staged)
  }
  return SCAPE_OK;
}

}  // namespace

extern "C" int scape_get(scape_t* h, int what, int r, void* buf, size_t bytes, void* cuda_stream) {
  if (!h || !buf) return fail(SCAPE_EINVAL, "NULL argument");
  DeviceGuard guard(h->dev);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  { const int jr = join_side(h, st); if (jr) return jr; }     // a refresh on the handle's own stream comes first
  const size_t nbytes = sizeof(float) * (size_t)h->N;
  MaskSlot& nx = h->slot[h->use];
  MaskSlot& la = h->slot[h->last];
  int rc = SCAPE_OK;
  switch (what) {
    case SCAPE_MOMENT:
      if (bytes != nbytes) return fail(SCAPE_EINVAL, "moment: expected %zu bytes", nbytes);
      if ((rc = materialise_dense_m(h, st))) return rc;      // dense view; the sparse store stays in use
      CU_TRY(cudaMemcpyAsync(buf, h->m, bytes, cudaMemcpyDefault, st));
      break;
    case SCAPE_RESIDUAL:
      if (r < 0 || r >= h->R) return fail(SCAPE_EINVAL, "residual: replica %d out of range", r);
      if (bytes != nbytes) return fail(SCAPE_EINVAL, "residual: expected %zu bytes", nbytes);
      CU_TRY(cudaMemcpyAsync(buf, h->e + (size_t)r * h->Npad, bytes, cudaMemcpyDefault, st));
      break;
    case SCAPE_MASK_NEXT:
    case SCAPE_MASK_LAST: {
      MaskSlot& s = what == SCAPE_MASK_NEXT ? nx : la;
      if (what == SCAPE_MASK_LAST && (h->t == 0 || !s.valid)) return fail(SCAPE_EINVAL, "no step has run yet");
      const size_t mb = sizeof(uint32_t) * (size_t)((h->N + 31) / 32);
      if (bytes != mb) return fail(SCAPE_EINVAL, "mask: expected %zu bytes", mb);
      if (s.all_ones && (rc = materialise_all_ones(h, s, st))) return rc;
      CU_TRY(cudaMemcpyAsync(buf, s.bits, bytes, cudaMemcpyDefault, st));
      break;
    }
    case SCAPE_IDX_NEXT:
      if ((rc = get_idx(h, nx, buf, bytes, st))) return rc;
      break;
    case SCAPE_IDX_LAST:
      if (h->t == 0 || !la.valid) return fail(SCAPE_EINVAL, "no step has run yet");
      if ((rc = get_idx(h, la, buf, bytes, st))) return rc;
      break;
    case SCAPE_PACKED: {
      if (h->t == 0 || !la.valid) return fail(SCAPE_EINVAL, "no step has run yet");
      if (r < 0 || r >= h->R) return fail(SCAPE_EINVAL, "packed: replica %d out of range", r);
      if (bytes != sizeof(float) * (size_t)la.count) return fail(SCAPE_EINVAL, "packed: expected %zu bytes", sizeof(float) * (size_t)la.count);
      if (h->last_dense) {
        if (!h->dense_pack) return fail(SCAPE_EINVAL, "packed: the last step's mask was all ones and keep_dense_pack is off");
        CU_TRY(cudaMemcpyAsync(buf, h->dense_pack + (size_t)r * h->Npad, bytes, cudaMemcpyDefault, st));
      } else {
        CU_TRY(cudaMemcpyAsync(buf, h->packed + (size_t)r * h->packed_stride, bytes, cudaMemcpyDefault, st));
      }
      break;
    }
    case SCAPE_PACKED_MEAN:
      if (h->t == 0 || !la.valid) return fail(SCAPE_EINVAL, "no step has run yet");
      if (bytes != sizeof(float) * (size_t)la.count) return fail(SCAPE_EINVAL, "packed_mean: expected %zu bytes", sizeof(float) * (size_t)la.count);
      CU_TRY(cudaMemcpyAsync(buf, h->last_dense ? h->m : h->pm[h->pm_last], bytes, cudaMemcpyDefault, st));
      break;
    default:
      return fail(SCAPE_EINVAL, "scape_get: bad selector %d", what);
  }
  CU_TRY(cudaStreamSynchronize(st));
  return SCAPE_OK;
}

extern "C" int scape_set(scape_t* h, int what, int r, const void* buf, size_t bytes, void* cuda_stream) {
  if (!h || !buf) return fail(SCAPE_EINVAL, "NULL argument");
  if (h->pending) return fail(SCAPE_EINVAL, "a split step is in flight: scape_step_apply first");
  DeviceGuard guard(h->dev);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  { const int jr = join_side(h, st); if (jr) return jr; }     // a refresh on the handle's own stream comes first
  const size_t nbytes = sizeof(float) * (size_t)h->N;
  switch (what) {
    case SCAPE_MOMENT:
      if (bytes != nbytes) return fail(SCAPE_EINVAL, "moment: expected %zu bytes", nbytes);
      CU_TRY(cudaMemcpyAsync(h->m, buf, bytes, cudaMemcpyDefault, st));
      h->m_sparse = false;                                   // m is dense again until the next sparse step
      break;
    case SCAPE_RESIDUAL:
      if (r < 0 || r >= h->R) return fail(SCAPE_EINVAL, "residual: replica %d out of range", r);
      if (bytes != nbytes) return fail(SCAPE_EINVAL, "residual: expected %zu bytes", nbytes);
      CU_TRY(cudaMemcpyAsync(h->e + (size_t)r * h->Npad, buf, bytes, cudaMemcpyDefault, st));
      break;
    case SCAPE_MASK_NEXT: {
      // The mask is validated in the `build` slot (free between steps: it holds M_{t-2}) and only
      // then becomes the `use` slot, so a refused mask leaves the handle as it was.
      MaskSlot& s = h->slot[h->build];
      const size_t mb = sizeof(uint32_t) * (size_t)((h->N + 31) / 32);
      if (bytes != mb) return fail(SCAPE_EINVAL, "mask: expected %zu bytes", mb);
      CU_TRY(cudaMemsetAsync(s.bits, 0, sizeof(uint32_t) * h->n_words, st));
      CU_TRY(cudaMemcpyAsync(s.bits, buf, bytes, cudaMemcpyDefault, st));
      mask_clear_tail_kernel<<<1, 256, 0, st>>>(s.bits, h->n_words, h->N);
      h->launches++;
      // count first (rank only), then decide whether an index list fits
      int rc = compact_mask(h, s, false, st);
      if (rc) return rc;
      uint32_t total = 0;
      CU_TRY(cudaMemcpyAsync(&total, h->total, sizeof total, cudaMemcpyDeviceToHost, st));
      CU_TRY(cudaStreamSynchronize(st));
      s.valid = false;
      if ((int64_t)total != h->N && (int64_t)total > h->packed_stride)
        return fail(SCAPE_EINVAL, "mask: %u bits set, at most %lld (the packed capacity) or all N allowed", total, (long long)h->packed_stride);
      if ((int64_t)total == h->N) {
        s.all_ones = true; s.count = h->N;
      } else {
        s.all_ones = false; s.count = total;
        if ((rc = compact_mask(h, s, true, st))) return rc;
      }
      s.valid = true;
      std::swap(h->use, h->build);
      break;
    }
    default:
      return fail(SCAPE_EINVAL, "scape_set: selector %d is not settable", what);
  }
  CU_TRY(cudaStreamSynchronize(st));
  return SCAPE_OK;
}

// ------------------------------------------------------------------------------------------
// scape_mask_indices_static: the ordered compaction of a bit mask (bits -> ascending int32 index
// list + count; stage 4's index half) for callers that cannot allocate: code under
// CUDA graph capture, serving loops, harnesses that forbid cudaMalloc.  A variant of
// mask_compact_kernel (single pass, chained scan with decoupled look-back) whose look-back state
// lives in a file-scope array of the library instead of a cudaMalloc'ed buffer of a handle.
// Every GPU that loads the library holds the array (kStaticScratchWords x 8 bytes = 33 KB) until
// the process exits.  All calls on one device share it: calls that overlap on the GPU race.
// ------------------------------------------------------------------------------------------
namespace {

constexpr int kStaticMaxBlocks = (int)(SCAPE_STATIC_MAX_BITS / ((int64_t)kCompactChunksPerBlock * 128));   // 4096 CTAs of 1024 chunks
static_assert((int64_t)kStaticMaxBlocks * kCompactChunksPerBlock * 128 == SCAPE_STATIC_MAX_BITS, "SCAPE_STATIC_MAX_BITS: whole blocks");
constexpr int kStaticCtlWord = kStaticMaxBlocks;          // [0, kStaticMaxBlocks): look-back state; then one word: {total, ticket}
constexpr int kStaticScratchWords = kStaticMaxBlocks + 32;
// In host code this name is a host-side stand-in, not a device address: static_scratch_ptr() resolves it per device.
static __device__ __align__(256) unsigned long long g_static_scratch[kStaticScratchWords];

constexpr int kMaxDevices = 64;
unsigned long long* g_static_scratch_addr[kMaxDevices] = {};
std::mutex g_static_mu;

// device address of g_static_scratch on device `dev`, which must be current; resolved once per device
int static_scratch_ptr(int dev, unsigned long long** out) {
  if (dev < 0 || dev >= kMaxDevices) return fail(SCAPE_EINVAL, "device ordinal %d out of range", dev);
  std::lock_guard<std::mutex> lock(g_static_mu);
  if (g_static_scratch_addr[dev] == nullptr) {
    void* p = nullptr;
    CU_TRY(cudaGetSymbolAddress(&p, g_static_scratch));
    if (p == nullptr) return fail(SCAPE_ECUDA, "cudaGetSymbolAddress returned a null address");
    g_static_scratch_addr[dev] = static_cast<unsigned long long*>(p);
  }
  *out = g_static_scratch_addr[dev];
  return SCAPE_OK;
}

// state[b] = (tag << 32) | value; tag 1: total of block b, 2: inclusive prefix through block b, 0 (cleared by the
// entry point before every launch): nothing yet.  ctl[0] = ticket.  One thread per chunk of 128 bits.
__global__ void __launch_bounds__(1024) mask_indices_static_kernel(const uint32_t* __restrict__ bits, int64_t n, int64_t n_words,
                                                                  int64_t n_chunks, unsigned long long* state, uint32_t* ctl,
                                                                  int32_t* __restrict__ idx, int64_t idx_cap, uint32_t* __restrict__ count_out) {
  __shared__ uint32_t ws[32];
  __shared__ uint32_t s_bid, s_prefix;
  if (threadIdx.x == 0) s_bid = atomicAdd(&ctl[0], 1u);     // ticket: every predecessor has started
  __syncthreads();
  const uint32_t bid = s_bid;
  const int64_t c = (int64_t)bid * kCompactChunksPerBlock + threadIdx.x;
  uint4 w = make_uint4(0, 0, 0, 0);
  if (c < n_chunks) {
    if ((c << 2) + 4 <= n_words && (c << 7) + 128 <= n) {
      w = __ldg(reinterpret_cast<const uint4*>(bits) + c);
    } else {                                                 // the ragged last chunk: word by word, bits at positions >= n ignored
      uint32_t x[4] = {0u, 0u, 0u, 0u};
      for (int q = 0; q < 4; ++q) {
        const int64_t wi = (c << 2) + q, lo = wi << 5;
        if (wi < n_words && lo < n) {
          x[q] = __ldg(bits + wi);
          if (lo + 32 > n) x[q] &= (1u << (uint32_t)(n - lo)) - 1u;
        }
      }
      w = make_uint4(x[0], x[1], x[2], x[3]);
    }
  }
  const uint32_t cnt = __popc(w.x) + __popc(w.y) + __popc(w.z) + __popc(w.w);
  uint32_t incl = cnt;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const uint32_t x = __shfl_up_sync(0xFFFFFFFFu, incl, o); if (lane >= o) incl += x; }
  if (lane == 31) ws[wid] = incl;
  __syncthreads();
  constexpr unsigned long long tag_total = 1ull << 32, tag_incl = 2ull << 32;
  if (wid == 0) {
    const uint32_t x = ws[lane];
    uint32_t ix = x;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const uint32_t y = __shfl_up_sync(0xFFFFFFFFu, ix, o); if (lane >= o) ix += y; }
    ws[lane] = ix - x;
    const uint32_t total = __shfl_sync(0xFFFFFFFFu, ix, 31);
    volatile unsigned long long* vs = state;
    if (lane == 0) { vs[bid] = (bid == 0 ? tag_incl : tag_total) | total; __threadfence(); }
    uint32_t prefix = 0;
    if (bid > 0) {
      int64_t b0 = (int64_t)bid - 1;                         // newest predecessor not yet accounted for
      while (true) {
        const int64_t b = b0 - lane;
        unsigned long long v = 0;
        bool ready, is_incl;
        do {                                                 // until every predecessor in the window has published
          v = b >= 0 ? vs[b] : tag_incl;                     // before block 0: an inclusive prefix of 0
          const unsigned long long tg = v & 0xFFFFFFFF00000000ull;
          is_incl = tg == tag_incl;
          ready = is_incl || tg == tag_total;
        } while (!__all_sync(0xFFFFFFFFu, ready));
        const uint32_t incl_mask = __ballot_sync(0xFFFFFFFFu, is_incl);
        const int stop = incl_mask ? __ffs(incl_mask) - 1 : 31;      // nearest predecessors first, up to the first inclusive one
        uint32_t val = lane <= stop ? (uint32_t)v : 0u;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) val += __shfl_xor_sync(0xFFFFFFFFu, val, o);
        prefix += val;
        if (incl_mask) break;
        b0 -= 32;
      }
      if (lane == 0) { __threadfence(); vs[bid] = tag_incl | (prefix + total); }
    }
    if (lane == 0) {
      s_prefix = prefix;
      if (bid == gridDim.x - 1) *count_out = prefix + total;
    }
  }
  __syncthreads();
  const uint32_t j = s_prefix + ws[wid] + incl - cnt;
  write_chunk_indices(w, cnt, j, c, idx, idx_cap);           // whole warps (past the end: w = 0, cnt = 0)
}

}  // namespace

extern "C" int scape_mask_indices_static(const uint32_t* mask_words, int64_t n, int32_t* idx_out, int64_t idx_cap,
                                         uint32_t* count_out, void* cuda_stream) {
  if (n < 0) return fail(SCAPE_EINVAL, "n must be >= 0");
  if (n > SCAPE_STATIC_MAX_BITS)
    return fail(SCAPE_EINVAL, "n = %lld exceeds SCAPE_STATIC_MAX_BITS = %lld (the static scratch array holds the state of %d blocks of 131072 bits)",
                (long long)n, (long long)SCAPE_STATIC_MAX_BITS, kStaticMaxBlocks);
  if (idx_cap < 0) return fail(SCAPE_EINVAL, "idx_cap must be >= 0");
  if (!count_out) return fail(SCAPE_EINVAL, "NULL count_out");
  if ((uintptr_t)count_out & 3) return fail(SCAPE_EINVAL, "count_out must be 4-byte aligned");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (n == 0) { CU_TRY(cudaMemsetAsync(count_out, 0, sizeof(uint32_t), st)); return SCAPE_OK; }
  if (!mask_words) return fail(SCAPE_EINVAL, "NULL mask_words");
  if ((uintptr_t)mask_words & 15) return fail(SCAPE_EINVAL, "mask_words must be 16-byte aligned");
  if (idx_cap > 0 && !idx_out) return fail(SCAPE_EINVAL, "NULL idx_out with idx_cap > 0");
  if ((uintptr_t)idx_out & 3) return fail(SCAPE_EINVAL, "idx_out must be 4-byte aligned");
  int dev = -1;
  CU_TRY(cudaGetDevice(&dev));
  unsigned long long* scratch = nullptr;
  int rc = static_scratch_ptr(dev, &scratch);
  if (rc) return rc;
  const int64_t n_words = (n + 31) >> 5;
  const int64_t n_chunks = (n + 127) >> 7;
  const int nb = (int)((n_chunks + kCompactChunksPerBlock - 1) / kCompactChunksPerBlock);
  // the array keeps the last call's contents: the state words of this call's blocks and the ticket start at zero
  CU_TRY(cudaMemsetAsync(scratch, 0, sizeof(unsigned long long) * (size_t)nb, st));
  CU_TRY(cudaMemsetAsync(scratch + kStaticCtlWord, 0, sizeof(unsigned long long), st));
  mask_indices_static_kernel<<<nb, 1024, 0, st>>>(mask_words, n, n_words, n_chunks, scratch,
                                                  reinterpret_cast<uint32_t*>(scratch + kStaticCtlWord),
                                                  idx_cap > 0 ? idx_out : nullptr, idx_cap, count_out);
  CU_TRY(cudaGetLastError());
  return SCAPE_OK;
}
