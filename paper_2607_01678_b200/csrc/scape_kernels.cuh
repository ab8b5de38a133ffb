// scape_kernels.cuh — sm_100a kernels of the SCAPE step (Algorithm 1, :131-174).
//
// Data layout: the shard is cut into CHUNKS of 128 consecutive
// parameters; one warp handles one chunk per loop trip, lane l owning elements 4l..4l+3
// (one 128-bit access per fp32 array, one 64-bit access per bf16 array).  A mask is stored as
// bits (word i/32, bit i%32 => one uint4 per chunk) plus position tables: `pre[c]`, the running
// popcounts of chunk c's four words, one byte each (byte 3 = the chunk's total); the number of set
// bits before the chunk ("rank128"); and `trank[T]`, the number of set bits before TILE T = chunks
// 8T .. 8T+7 (the 8 chunks the warps of one CTA handle together).  The packed position of a selected
// element is rank128 + words before + popc(bits before it inside its word): the pack of Alg. 1 l.9
// needs no atomics and keeps ascending index order, and a lane finds its position from ONE word of
// bits and the chunk's table entry (no popcounts over other words).  Two views of the tables exist:
//   rk[c] = {rank128, pre}   8 bytes per chunk: one load, a handful of instructions; the register-
//                            staged kernel (issue- and register-bound) and every other kernel use it
//   pre[c] + trank[T]        4 bytes per chunk + 4 per tile; rank128 = trank + the totals of the
//                            tile's earlier chunks (one shuffle, one warp-wide add).  The bulk-copy
//                            staged kernel is HBM-bound and uses this one: rk was 3.5 M more 32-byte
//                            sector reads per step on the headline shard and cost that kernel 0.2 ms
//                            (1.5 % for 0.13 % of the bytes: small reads between the streams' bursts
//                            are dear).
//
// Every fp32 operation of the method is written with a _rn intrinsic so that nvcc cannot
// contract or reorder it; the order is the one pinned in DESIGN.md and followed by the oracle.
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace scapek {

constexpr int kChunk = 128;          // parameters per warp trip
constexpr int kMaxR = 8;
constexpr int kDigitBits = 13;       // radix-select digit width
constexpr int kBins = 1 << kDigitBits;
constexpr int kSelPasses = 5;        // 64-bit composite key = 13+13+13+13+12 bits

// Predicted threshold bracket of one top-k problem (the flat partition, or one layer): in the coming
// step's fused pass key >= hi_key is certainly selected, lo_key <= key < hi_key is a candidate,
// key < lo_key is certainly not selected.  lo_key = hi_key = 0xFFFFFFFF: nothing predicted.
struct Bracket {
  uint32_t lo_key, hi_key;
  float delta;                // half-width of the bracket in ln(threshold)
  float lnT_prev;             // ln of the last exact threshold |m~| value
  float ln_pred;              // ln of the threshold that was predicted for the current step
  float r_prev;               // previous step-to-step change of ln(threshold)
  int have_T;                 // number of exact thresholds seen (saturates at 2)
};

// Device-resident control block of the stage-2 select (never read by the host on the timed path).
struct SelState {
  unsigned long long prefix;  // digits of T64 fixed so far
  unsigned long long himask;  // mask of those digits
  long long rank;             // rank (1-based from the top) still sought inside the prefix class
  int top;                    // bits [0, top) of K64 are still undecided; 0 = T64 is complete
  int use_cls;                // the surviving class has been collected into the small list
  unsigned long long class_count;   // keys in the class chosen by the last pick
  unsigned int cls_n;         // entries in the small list
  unsigned int first_bits;    // > 0: the histogram of the first digit (this many bits) is already in ghist: the streaming kernel made it
  unsigned long long base;    // fast route: the radix passes run on K64 - base (base = lo_key << 32), see sel_decide_kernel
  Bracket br;                 // predicted bracket for the COMING step's fused pass
  unsigned long long cand_cap_total;   // n_seg * seg_cap of the last fused pass
  int hit;                    // this step: 1 = the bracket held (candidate list), 0 = general path
  unsigned long long n_fast, n_general;   // statistics (scape_select_stats)
  unsigned long long n_above, n_cand;     // this step's counts from the fused pass
  // Recovery of a missed bracket (and the select of an all-ones step): a bracket taken from a sampled
  // histogram, one classification pass over every key, then the candidate route (sel_sample_kernel ...)
  int need_rec;               // this step: the predicted bracket missed (or there was none): the recovery kernels run
  int rec;                    // this step: the candidate list is the recovery pass's (its own segment layout, bracket [lo2, hi2))
  uint32_t lo2, hi2;
  unsigned long long n_recovered;         // statistics: steps the recovery pass saved from the general route
  int bits_done;              // candidate route: the pass that collected the surviving class also set the bits of every candidate
                              // above that class, so sel_finish_kernel only has the small list left to look at
};

// Per-layer top-k (PAPER.md:89 "per-layer style", :138): one of these per layer, device-resident.
struct LayerState {
  long long begin, end;       // the layer is [begin, end) of the flattened shard
  long long k;                // entries the current refresh selects in this layer (end - begin when not compressed)
  int compress;               // 0: never sparsified (LayerNorm, RMSNorm, bias: PAPER.md:246, :279, :286)
  int hit;                    // this step: 1 = the layer's bracket held (candidate list), 0 = general route
  unsigned long long prefix;  // digits of the layer's T64 fixed so far
  unsigned long long himask;
  long long rank;
  int top;                    // bits [0, top) of K64 still undecided; 0 = T64 complete
  int skip;                   // workers: another worker makes this layer's mask (scape_set_workers); no bit is set here
  unsigned long long n_above; // certainly-selected entries counted by the fused pass (reset by lsel_decide)
  unsigned long long base;    // candidate route: the radix passes run on K64 - base (base = lo_key << 32); 0 otherwise
  Bracket br;
};

// Control block of the per-layer select.
struct LayerCtl {
  int any_general;            // some layer takes the general route in this step
  int overflow;               // a candidate segment overflowed: every compressed layer goes general
  float shrink;               // > 0: the candidate list was more than half full, narrow every bracket
  int pad;
  unsigned long long n_fast, n_general;   // layer-steps on each route (statistics)
  // small list: once the surviving classes of all candidate-route layers together hold at most
  // kClsCap keys, the next pass copies them out and the remaining passes read only that list
  unsigned long long cls_total; // keys in the classes the last picks chose (candidate-route layers)
  unsigned int cls_n;           // entries in the small list
  int use_cls;                  // the small list is complete: read it instead of the segments
  int bits_done;                // the collecting pass also set the bits of the candidates above their layer's class (see SelState)
};

struct StepParams {
  float* theta;                 // [N] caller-owned
  float* m;                     // [Npad]
  float* e;                     // [R][e_stride]
  int64_t e_stride;
  const void* g[kMaxR];         // R caller-owned gradient buffers
  const uint32_t* cur_bits;     // [Npad/32]   (unused when DENSE)
  const uint2* cur_rk;          // [Npad/128] {set bits before the chunk, its word prefixes}: register-staged kernel
  const uint32_t* cur_pre;      // [8 * n_tiles] word prefixes of every chunk (see chunk_prefix_bytes): staged kernel
  const uint32_t* cur_trank;    // [n_tiles + 1] set bits before every tile of 8 chunks (last entry: all of them)
  float* packed;                // [R][packed_stride] or nullptr (DENSE without keep_dense_pack)
  int64_t packed_stride;
  float* packed_mean;           // [k] b- of this step = m_t in packed form (unused when DENSE)
  // m_{t-1} stored sparsely (MSPARSE): it is zero off the mask the previous step used (Eq. 4,
  // PAPER.md:197), so it lives as that step's packed mean, addressed through that mask
  const uint32_t* prev_bits;    // [Npad/32]
  const uint2* prev_rk;         // [Npad/128]
  const uint32_t* prev_pre;     // [8 * n_tiles]
  const uint32_t* prev_trank;   // [n_tiles + 1]
  const float* pm_prev;         // [k]
  int64_t N;
  int64_t n_chunks;             // ceil(N/128)
  // Sub-range launches (scape_step_host pipelines upload / step / download part by part): this launch covers
  // chunks [c_begin, c_end) -- multiples of 8 except c_end = n_chunks -- and its warps use the candidate
  // segments from seg_base on.  A whole-shard launch: 0, n_chunks, 0.  (Not in the grouped staged kernel.)
  uint32_t c_begin, c_end, seg_base;
  float b1, c1, b2, c2, eps, wd, neg_lr;
  float R_f, inv_R;
  int r_pow2;
  float bc1, bc2;               // bias-correction factors 1/(1-beta^t); 1.0f when off
  // l.14 clip_grad (optional): the pass stores g^ and beta2*m^2 of every selected entry, sums g^^2
  // in double, and leaves theta on the mask alone; clip_update_kernel finishes l.14-17 there
  // clip = 2 (workers, scape_step_local): the mean of l.10 needs the other workers' sums first, so
  // the pass parks the LOCAL sum over its replicas in ghat and m_old in vm, and leaves theta on the
  // mask to dist_update_kernel (scape_step_apply), which runs after the all-reduce
  int clip;
  float* ghat;                  // [K] packed
  float* vm;                    // [K] packed
  double* sumsq;                // one slot per warp of the launch
  int stash;                    // DENSE only: leave m~^0 in e^0 (keys for the select), not 0
  // stage 2 fused into the pass (sparse variant only)
  const SelState* ctl;          // bracket predicted by the previous step
  uint32_t* fused_hist;         // register-staged kernel, flat top-k: histogram of the candidates' first radix digit (kFusedBits
                                // bits), added to these global counters at the end of the kernel; nullptr: not wanted
  uint32_t* next_bits;          // [Npad/32] certainly-selected bits of M_t (complete overwrite)
  unsigned long long* cand;     // [n_seg][seg_cap] candidate composite keys, one segment per warp
  uint32_t* seg_count;          // [n_seg] candidates this warp saw (may exceed seg_cap: overflow)
  uint32_t* seg_above;          // [n_seg] certainly-selected entries this warp saw
  uint32_t seg_cap;
  // per-layer refresh (nullptr = one flat top-k): layer of each chunk's first element, bit 31 set
  // when the chunk holds entries of more than one layer
  const uint32_t* chunk_layer;  // [Npad/128]
  LayerState* layers;
};

// ------------------------------------------------------------------------------------------
// 128-bit streaming accesses.  ld.global.cs / st.global.cs = evict-first: every dense array is
// touched exactly once per step, so nothing here should displace the small resident arrays
// (mask bits, rank128, packed buffers) from L2.
// ------------------------------------------------------------------------------------------
template <bool GUARD>
__device__ __forceinline__ void load4_f32(const float* __restrict__ p, uint32_t i0, int64_t N, float (&v)[4]) {
  if (!GUARD) {
    const float4 t = __ldcs(reinterpret_cast<const float4*>(p + i0));
    v[0] = t.x; v[1] = t.y; v[2] = t.z; v[3] = t.w;
  } else {
#pragma unroll
    for (int q = 0; q < 4; ++q) v[q] = (i0 + q < N) ? __ldcs(p + i0 + q) : 0.0f;
  }
}

template <bool GUARD>
__device__ __forceinline__ void store4_f32(float* __restrict__ p, uint32_t i0, int64_t N, const float (&v)[4]) {
  if (!GUARD) {
    __stcs(reinterpret_cast<float4*>(p + i0), make_float4(v[0], v[1], v[2], v[3]));
  } else {
#pragma unroll
    for (int q = 0; q < 4; ++q) if (i0 + q < N) __stcs(p + i0 + q, v[q]);
  }
}

// Gradient loads: fp32, or bf16 widened exactly (S16) by placing the 16 bits in the high half.
template <typename G, bool GUARD>
__device__ __forceinline__ void load4_grad(const void* __restrict__ base, uint32_t i0, int64_t N, float (&v)[4]) {
  if constexpr (sizeof(G) == 4) {
    load4_f32<GUARD>(reinterpret_cast<const float*>(base), i0, N, v);
  } else {
    const uint16_t* p = reinterpret_cast<const uint16_t*>(base);
    if (!GUARD) {
      const uint2 t = __ldcs(reinterpret_cast<const uint2*>(p + i0));
      v[0] = __uint_as_float(t.x << 16); v[1] = __uint_as_float(t.x & 0xFFFF0000u);
      v[2] = __uint_as_float(t.y << 16); v[3] = __uint_as_float(t.y & 0xFFFF0000u);
    } else {
#pragma unroll
      for (int q = 0; q < 4; ++q)
        v[q] = (i0 + q < N) ? __uint_as_float(((uint32_t)__ldcs(p + i0 + q)) << 16) : 0.0f;
    }
  }
}

// Position of this lane's 4 mask bits inside the chunk's uint4, and the packed rank before them.
__device__ __forceinline__ void lane_bits_from_words(const uint4 mw, const uint32_t r0, int lane, uint32_t& mybits, uint32_t& jbase) {
  const int ws = lane >> 3, sh = (lane & 7) << 2;
  const uint32_t p0 = __popc(mw.x), p1 = p0 + __popc(mw.y), p2 = p1 + __popc(mw.z);
  const uint32_t w = ws == 0 ? mw.x : ws == 1 ? mw.y : ws == 2 ? mw.z : mw.w;
  const uint32_t before = ws == 0 ? 0u : ws == 1 ? p0 : ws == 2 ? p1 : p2;
  mybits = (w >> sh) & 0xFu;
  jbase = r0 + before + __popc(w & ((1u << sh) - 1u));
}
__device__ __forceinline__ uint32_t chunk_popc(const uint4 mw) { return __popc(mw.x) + __popc(mw.y) + __popc(mw.z) + __popc(mw.w); }

// pre[c]: running popcounts of the chunk's words, one byte each (byte 3 = the chunk's total, <= 128)
__host__ __device__ __forceinline__ uint32_t chunk_prefix_bytes(uint32_t p0, uint32_t p1, uint32_t p2, uint32_t p3) {
  return p0 | ((p0 + p1) << 8) | ((p0 + p1 + p2) << 16) | ((p0 + p1 + p2 + p3) << 24);
}

// Where a lane's 4 mask bits sit: word ws of the chunk, bits sh..sh+3.  Loop-invariant per lane, so the
// streaming kernels decode a chunk's mask with one 32-bit load of the lane's OWN word, the tile's 8
// `pre` words (lane l loads word l % 8), trank (same address for the whole warp), one shuffle, one
// warp-wide add, a byte pick (PRMT), a shift, two ANDs and one POPC.
struct LaneMap { uint32_t ws, sh, lowmask, sel; };
__device__ __forceinline__ LaneMap lane_map(int lane) {
  LaneMap lm;
  lm.ws = (uint32_t)lane >> 3; lm.sh = ((uint32_t)lane & 7u) << 2;
  lm.lowmask = (1u << lm.sh) - 1u;
  lm.sel = lm.ws == 0 ? 0x4444u : 0x4440u + (lm.ws - 1u);      // __byte_perm selector: byte ws-1 of rk.y, or 0
  return lm;
}
__device__ __forceinline__ void lane_decode(uint32_t w, uint2 rk, const LaneMap& lm, uint32_t& mybits, uint32_t& jbase) {
  mybits = (w >> lm.sh) & 0xFu;
  jbase = rk.x + __byte_perm(rk.y, 0u, lm.sel) + __popc(w & lm.lowmask);
}
// {set bits before chunk `pos` of its tile, the chunk's own prefix word} from what the warp holds:
// pa = pre[8T + lane % 8], tr = trank[T].  Whole warps only (one shuffle, one warp-wide add).
__device__ __forceinline__ uint2 chunk_rank(uint32_t pa, uint32_t tr, uint32_t pos, int lane) {
  const uint32_t mine = __shfl_sync(0xFFFFFFFFu, pa, (int)pos);
  const uint32_t before = __reduce_add_sync(0xFFFFFFFFu, (uint32_t)lane < pos ? pa >> 24 : 0u);
  return make_uint2(tr + before, mine);
}
// a lane's 4 mask bits of chunk c and the packed position of the first of them
__device__ __forceinline__ void lane_mask_bits(const uint32_t* __restrict__ bits, const uint2* __restrict__ rk,
                                               int64_t c, int lane, uint32_t& mybits, uint32_t& jbase) {
  const uint4 mw = __ldg(reinterpret_cast<const uint4*>(bits) + c);
  lane_bits_from_words(mw, __ldg(rk + c).x, lane, mybits, jbase);
}

// Gather of m_{t-1} for this lane's 4 elements from the previous step's packed mean: selected
// entries sit at consecutive packed positions from pbase on, so one pointer walks them.
__device__ __forceinline__ void gather_prev_m(const float* __restrict__ pm, uint32_t pbits, uint32_t pbase, float (&mo)[4]) {
  const float* ptr = pm + pbase;
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    const bool on = (pbits >> q) & 1u;
    mo[q] = on ? __ldg(ptr) : 0.0f;
    ptr += on ? 1 : 0;
  }
}

// ------------------------------------------------------------------------------------------
// Stages 1, 3, 4, 5, 6 fused: one streaming pass (Alg. 1 l.6-10, l.12-17).
// ------------------------------------------------------------------------------------------
struct StageA {                 // per-warp running state of the fused select (registers)
  uint32_t lo, hi;              // bracket keys
  uint32_t n_above;             // per lane
  uint32_t cursor;              // warp-uniform: candidates appended so far
  unsigned long long* seg;      // this warp's candidate segment
  double sumsq;                 // per lane: sum of g^^2 (clip mode)
  uint32_t layer;               // per-layer refresh: layer whose bracket is loaded (kNoLayer: none yet)
};
constexpr uint32_t kNoLayer = 0xFFFFFFFFu;

// per-layer refresh: add this warp's count of certainly-selected entries to its layer
__device__ __forceinline__ void warp_flush_layer(const StepParams& p, StageA& sa, int lane) {
  uint32_t na = sa.n_above;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) na += __shfl_xor_sync(0xFFFFFFFFu, na, o);
  if (lane == 0 && na != 0u && sa.layer != kNoLayer) atomicAdd(&p.layers[sa.layer].n_above, (unsigned long long)na);
  sa.n_above = 0;
}

// clip mode: this warp's share of sum g^^2, lanes added in a fixed butterfly order
__device__ __forceinline__ void warp_store_sumsq(const StepParams& p, const StageA& sa, int64_t slot, int lane) {
  double v = sa.sumsq;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, o);
  if (lane == 0) p.sumsq[slot] = v;
}

// The arithmetic of one lane's 4 elements (Alg. 1 l.6-10, l.12-17 in the pinned order), the stores
// of theta / m / e^r / b^r / b-, and the bracket classification of stage 2.  Shared by the two
// load front-ends (register-staged LDG and shared-memory-staged bulk copies).

// All-ones mask (step 1, sparsity 0): dense m in and out, nothing is packed, no classification.
template <int R, bool GUARD, bool CLIPT>
__device__ __forceinline__ void dense_compute(const StepParams& p, uint32_t i0, float (&th)[4], const float (&mo)[4],
                                              float (&gg)[R][4], float (&ee)[R][4], StageA& sa) {
  float mn[4];
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    const float pq = __fmul_rn(p.b1, mo[q]);                // beta1 * m_{t-1}, reused by l.6 and l.13
    float mt[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
      mt[r] = __fadd_rn(__fmaf_rn(p.c1, gg[r][q], pq), ee[r][q]);            // l.6
      ee[r][q] = (r == 0 && p.stash) ? mt[r] : 0.0f;                         // l.8 (M = 1); stash: keys for the select
    }
    if (p.packed != nullptr && (!GUARD || i0 + q < p.N)) {
#pragma unroll
      for (int r = 0; r < R; ++r) p.packed[r * p.packed_stride + (i0 + q)] = mt[r];   // l.9 (keep_dense_pack)
    }
    float s = mt[0];
#pragma unroll
    for (int r = 1; r < R; ++r) s = __fadd_rn(s, mt[r]);                                   // l.10, r ascending
    const float bb = p.r_pow2 ? __fmul_rn(s, p.inv_R) : __fdiv_rn(s, p.R_f);              // l.10
    const float gh = __fdiv_rn(__fsub_rn(bb, pq), p.c1);                                    // l.13 (Eq. 3)
    const float vmq = __fmul_rn(p.b2, __fmul_rn(mo[q], mo[q]));
    mn[q] = bb;                                                                             // l.12
    if (CLIPT) {                                          // the CLIPT instantiations run with p.clip != 0 only (launch_fused)
      // l.14 needs the norm of g^ over the whole mask first: park what l.15-17 need; theta of
      // this entry is updated by clip_update_kernel
      if (!GUARD || i0 + q < p.N) {
        if (p.clip == 2) { p.ghat[i0 + q] = s; p.vm[i0 + q] = mo[q]; }
        else {
          p.ghat[i0 + q] = gh; p.vm[i0 + q] = vmq;
          sa.sumsq += (double)gh * (double)gh;
        }
      }
    } else {
      const float v = __fmaf_rn(p.c2, __fmul_rn(gh, gh), vmq);                              // l.15
      const float u = __fdiv_rn(__fmul_rn(bb, p.bc1), __fadd_rn(__fsqrt_rn(__fmul_rn(v, p.bc2)), p.eps));   // l.16 (+ :77)
      const float w = __fmaf_rn(p.wd, th[q], u);                                            // l.17
      th[q] = __fmaf_rn(p.neg_lr, w, th[q]);
    }
  }
  store4_f32<GUARD>(p.theta, i0, p.N, th);
#pragma unroll
  for (int r = 0; r < R; ++r) store4_f32<false>(p.e + r * p.e_stride, i0, p.N, ee[r]);
  store4_f32<false>(p.m, i0, p.N, mn);                    // sparse steps keep m_t as b- only
}

// Candidate keys of the register-staged front-end are staged in a per-warp shared-memory ring and
// leave for the warp's segment in global memory 32 at a time (one 256-byte store per warp): a lane
// with candidates takes its ring positions with ONE shared-memory atomic (no votes, no prefix over
// the lanes; the order inside a segment is irrelevant, the composite keys carry the index).
// The ring holds the < 32 keys not yet flushed plus the <= 128 a chunk can add.
constexpr uint32_t kRing = 256;
struct CandRing {
  unsigned long long* ring;     // [kRing] shared memory, private to the warp
  uint32_t* head;               // keys appended so far (shared memory); StageA::cursor = keys flushed so far
  uint32_t* hist;               // [1 << kFusedBits] shared memory of the CTA, or nullptr: first-digit histogram of the candidates
  uint32_t hist_shift;          // digit = (key - lo) >> hist_shift
};
// First radix digit of the candidate route, made on the fly (the radix-histogram select's first pass over the
// candidate list costs a third of the select stage at 90 % sparsity): every candidate key lies in [lo, hi), the
// passes run on K64 - (lo << 32) from bit top = 32 + bits(hi - 1 - lo) down (sel_decide_kernel), so a first
// digit of kFusedBits bits is (key - lo) >> (top - 32 - kFusedBits) -- usable when that shift is >= 0 and the
// remaining bits fit the remaining passes.
constexpr int kFusedBits = 10;
__host__ __device__ __forceinline__ int fused_hist_shift(uint32_t lo, uint32_t hi) {       // < 0: not usable
  if (lo == 0xFFFFFFFFu && hi == 0xFFFFFFFFu) return -1;
  const uint32_t span1 = hi - 1u - lo;
  int b = 0;
  while (b < 32 && (span1 >> b) != 0u) ++b;                   // bits of the largest key - lo
  if (b < kFusedBits || 32 + b - kFusedBits > kDigitBits * (kSelPasses - 1)) return -1;
  return b - kFusedBits;
}

__device__ __forceinline__ void ring_flush32(const StepParams& p, StageA& sa, const CandRing& cr, int lane) {
  const uint32_t j = sa.cursor + (uint32_t)lane;
  const unsigned long long v = cr.ring[j & (kRing - 1u)];
  if (j < p.seg_cap) sa.seg[j] = v;                         // a full segment drops keys; seg_count still counts them (overflow)
  if (cr.hist != nullptr) atomicAdd(&cr.hist[((uint32_t)(v >> 32) - sa.lo) >> cr.hist_shift], 1u);
  sa.cursor += 32u;
}
// end of the kernel: the < 32 keys still in the ring; returns the number of keys the warp appended
__device__ __forceinline__ uint32_t ring_drain(const StepParams& p, StageA& sa, const CandRing& cr, int lane) {
  __syncwarp();
  const uint32_t head = *reinterpret_cast<volatile uint32_t*>(cr.head);
  while (head - sa.cursor >= 32u) ring_flush32(p, sa, cr, lane);
  const uint32_t j = sa.cursor + (uint32_t)lane;
  if (j < head) {
    const unsigned long long v = cr.ring[j & (kRing - 1u)];
    if (j < p.seg_cap) sa.seg[j] = v;
    if (cr.hist != nullptr) atomicAdd(&cr.hist[((uint32_t)(v >> 32) - sa.lo) >> cr.hist_shift], 1u);
  }
  return head;
}

// Sparse mask.  The selected entries of a chunk (cnt of 128; ~13 at 90 % sparsity, ~1 at 99 %) are
// scattered over the lanes, so running l.10-16 (IEEE divisions, square root) where they sit would
// mean four divergent passes with a few active lanes each, and b^r would leave as scattered 4-byte
// stores.  Instead every lane parks (m_old, m~^0 .. m~^{R-1}) of its selected entries in a
// warp-private scratch at the entry's rank inside the chunk, and lane l then handles the entry of
// rank l: b^r (l.9), b- (l.10, l.12) stored coalesced, l.13-16 in one pass over consecutive lanes.
// The update u comes back through the same scratch.
//   r0 = rank128[c]; cnt = set bits of the chunk
//   scm = 128 floats (m_old), sc = R arrays of 128 floats SCS floats apart (m~^r), private to this warp
//   RING: candidates go through the shared-memory ring `cr` (register-staged front-end), else straight
//   to the segment with one ballot per element (bulk-copy front-end: register-bound, shared memory full)
template <int R, bool GUARD, bool STORE, bool CLIPT, bool RING, int SCS>
__device__ __forceinline__ void sparse_compute(const StepParams& p, uint32_t c, int lane, const LaneMap& lm, uint32_t i0,
                                               uint32_t mybits, uint32_t jbase, uint32_t r0, uint32_t cnt, float* scm, float* sc,
                                               float (&th)[4], const float (&mo)[4],
                                               float (&gg)[R][4], float (&ee)[R][4], StageA& sa, const CandRing& cr) {
  uint32_t key0[4];             // bits(|m~^0|): the selection statistic of l.11
  constexpr bool deferred = CLIPT;                        // (p.clip != 0 there) theta on the mask is left to clip_update_kernel / dist_update_kernel
  if (cnt == 0) {
    // no selected entry in this chunk (88 % of the chunks at 99.9 % sparsity): l.6-8 and l.17 only
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      const float pq = __fmul_rn(p.b1, mo[q]);
#pragma unroll
      for (int r = 0; r < R; ++r) ee[r][q] = __fadd_rn(__fmaf_rn(p.c1, gg[r][q], pq), ee[r][q]);   // l.6-7
      key0[q] = __float_as_uint(ee[0][q]) & 0x7FFFFFFFu;
      th[q] = __fmaf_rn(p.neg_lr, __fmaf_rn(p.wd, th[q], 0.0f), th[q]);                            // l.17, u = 0 (Eq. 5)
    }
  } else {
    const uint32_t lbase = jbase - r0;                    // rank of this lane's first entry inside the chunk
    {
      float* ps = sc + lbase;                             // walks this lane's selected entries
      float* pm = scm + lbase;
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const bool on = (mybits >> q) & 1u;
        const float pq = __fmul_rn(p.b1, mo[q]);
        float mt[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
          mt[r] = __fadd_rn(__fmaf_rn(p.c1, gg[r][q], pq), ee[r][q]);            // l.6
          ee[r][q] = on ? 0.0f : mt[r];                                          // l.7-8
        }
        key0[q] = __float_as_uint(mt[0]) & 0x7FFFFFFFu;
        if (on) {
          *pm = mo[q];
#pragma unroll
          for (int r = 0; r < R; ++r) ps[r * SCS] = mt[r];
          ++ps; ++pm;
        }
      }
    }
    __syncwarp();
    for (uint32_t l = lane; l < cnt; l += 32) {           // lane l: the chunk's selected entry of rank l
      const float mq = scm[l];
      float sm = sc[l];
      float* pk = p.packed + (r0 + l);
      __stcs(pk, sm);                                                                       // l.9, r = 0
#pragma unroll
      for (int r = 1; r < R; ++r) {
        const float v = sc[r * SCS + l];
        pk += p.packed_stride;
        __stcs(pk, v);                                                                      // l.9
        sm = __fadd_rn(sm, v);                                                              // l.10, r ascending
      }
      const float pq = __fmul_rn(p.b1, mq);
      const float bb = p.r_pow2 ? __fmul_rn(sm, p.inv_R) : __fdiv_rn(sm, p.R_f);          // l.10
      const float gh = __fdiv_rn(__fsub_rn(bb, pq), p.c1);                                  // l.13 (Eq. 3)
      const float vmq = __fmul_rn(p.b2, __fmul_rn(mq, mq));
      p.packed_mean[r0 + l] = bb;                                                           // l.12: m_t = b-
      if (deferred) {
        if (p.clip == 2) { p.ghat[r0 + l] = sm; p.vm[r0 + l] = mq; }
        else {
          p.ghat[r0 + l] = gh; p.vm[r0 + l] = vmq;
          sa.sumsq += (double)gh * (double)gh;
        }
      } else {
        const float v = __fmaf_rn(p.c2, __fmul_rn(gh, gh), vmq);                            // l.15
        sc[l] = __fdiv_rn(__fmul_rn(bb, p.bc1), __fadd_rn(__fsqrt_rn(__fmul_rn(v, p.bc2)), p.eps));   // l.16 (+ :77)
      }
    }
    __syncwarp();
    {
      const float* pu = sc + lbase;
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const bool on = (mybits >> q) & 1u;
        const float u = on ? *pu : 0.0f;                                                     // Eq. 5 off the mask
        pu += on ? 1 : 0;
        if (deferred && on) continue;
        th[q] = __fmaf_rn(p.neg_lr, __fmaf_rn(p.wd, th[q], u), th[q]);                       // l.17
      }
    }
    __syncwarp();                                         // the scratch is reused by the next chunk
  }

  if (STORE) {                                            // else the caller stores th / ee (staged bulk stores)
    store4_f32<GUARD>(p.theta, i0, p.N, th);
#pragma unroll
    for (int r = 0; r < R; ++r) store4_f32<false>(p.e + r * p.e_stride, i0, p.N, ee[r]);
  }

  // Stage 2 (l.11) fused: classify |m~^0| against the predicted bracket.  Exactness does not
  // depend on the prediction: sel_decide_kernel checks n_above < k <= n_above + n_cand.
  bool mixed = false;                                     // chunk with entries of several layers (warp-uniform)
  if (p.chunk_layer != nullptr) {
    // per-layer refresh: the bracket is the one of this chunk's layer.  Warps walk the shard in
    // ascending order, so a layer change is rare: flush the count, load the new bracket.
    const uint32_t cl = __ldg(p.chunk_layer + c);
    const uint32_t l = cl & 0x7FFFFFFFu;
    mixed = (cl >> 31) != 0u;
    if (l != sa.layer) {
      warp_flush_layer(p, sa, lane);
      sa.layer = l;
      sa.lo = p.layers[l].br.lo_key; sa.hi = p.layers[l].br.hi_key;
    }
  }
  uint32_t nib = 0, cnib = 0;
  if (!mixed) {
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      const bool valid = !GUARD || (i0 + q < p.N);
      const bool above = valid && key0[q] >= sa.hi;
      nib |= above ? (1u << q) : 0u;
      cnib |= (valid && !above && key0[q] >= sa.lo) ? (1u << q) : 0u;
    }
  } else {
    // a chunk shared by several layers (at most one per layer boundary): bracket and count per entry
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      if (GUARD && i0 + q >= p.N) continue;
      uint32_t l = sa.layer;
      while (i0 + q >= p.layers[l].end) ++l;
      if (key0[q] >= p.layers[l].br.hi_key) { nib |= 1u << q; atomicAdd(&p.layers[l].n_above, 1ull); }
      else if (key0[q] >= p.layers[l].br.lo_key) cnib |= 1u << q;
    }
  }
  // Append this chunk's candidates (their order inside the segment is irrelevant: the composite
  // keys carry the index).
  if constexpr (RING) {
    if (cnib != 0u) {
      uint32_t pos = atomicAdd(cr.head, (uint32_t)__popc(cnib));
      const uint32_t inv = 0xFFFFFFFFu - (uint32_t)i0;
      uint2* ring2 = reinterpret_cast<uint2*>(cr.ring);
#pragma unroll
      for (int q = 0; q < 4; ++q)
        if ((cnib >> q) & 1u) { ring2[pos & (kRing - 1u)] = make_uint2(inv - q, key0[q]); ++pos; }   // little endian: low word = index part
    }
    __syncwarp();
    const uint32_t head = *reinterpret_cast<volatile uint32_t*>(cr.head);
    while (head - sa.cursor >= 32u) ring_flush32(p, sa, cr, lane);
  } else {
    if (__any_sync(0xFFFFFFFFu, cnib != 0u)) {              // candidates are rare here: usually skipped
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const bool cnd = (cnib >> q) & 1u;
        const uint32_t bal = __ballot_sync(0xFFFFFFFFu, cnd);
        if (cnd) {
          const uint32_t pos = sa.cursor + __popc(bal & ((1u << lane) - 1u));
          if (pos < p.seg_cap)
            sa.seg[pos] = ((unsigned long long)key0[q] << 32) | (unsigned long long)(0xFFFFFFFFu - (uint32_t)(i0 + q));
        }
        sa.cursor += __popc(bal);
      }
    }
  }
  if (!mixed) sa.n_above += __popc(nib);
  // the word of M_t this lane's group of 8 shares: OR of the nibbles (a REDUX per group of 8 lanes
  // compiles to four serialised collectives: slower than three shuffles)
  uint32_t w = nib << lm.sh;
  w |= __shfl_xor_sync(0xFFFFFFFFu, w, 1);
  w |= __shfl_xor_sync(0xFFFFFFFFu, w, 2);
  w |= __shfl_xor_sync(0xFFFFFFFFu, w, 4);
  if (lm.sh == 0u) p.next_bits[(c << 2) + lm.ws] = w;
}

// A chunk's mask words as one lane needs them: its own word of the current (and, MSPARSE, the previous) mask + rk[c]
struct MaskWords { uint32_t cw, pw; uint2 crk, prk; };        // own word of bits + rk[c]: current / previous mask
template <bool CUR, bool PREV>
__device__ __forceinline__ void load_mask_words(const StepParams& p, uint32_t c, const LaneMap& lm, MaskWords& w) {
  if (CUR) { w.cw = __ldg(p.cur_bits + (c << 2) + lm.ws); w.crk = __ldg(p.cur_rk + c); }
  if (PREV) { w.pw = __ldg(p.prev_bits + (c << 2) + lm.ws); w.prk = __ldg(p.prev_rk + c); }
}
// Which mask words the register-staged kernel fetches one trip ahead: 2 = both masks' (R = 1: 6 more live
// registers still fit the 48 of five CTAs per SM, step_ctas_per_sm), 1 = the previous mask's only (they feed the gather of m),
// 0 = none (R >= 3: the registers are worth more to the streaming loads; measured)
__host__ __device__ constexpr int step_prefetch(int R) { return R == 1 ? 2 : R == 2 ? 1 : 0; }

// One chunk of the register-staged front-end.  sc: this warp's scratch, (R + 1) x 128 floats.
// mw: this chunk's mask words, fetched during the previous trip (their L2 latency would otherwise sit
// in front of the gather of m and, as ptxas schedules it, of the streaming loads too: 23 % of the
// stall samples at R = 1); c_next: the chunk whose words to fetch now (0xFFFFFFFF: none).
template <typename G, int R, bool DENSE, bool MSPARSE, bool GUARD, bool CLIPT, bool RING, int PF>
__device__ __forceinline__ void fused_chunk(const StepParams& p, uint32_t c, uint32_t c_next, int lane, const LaneMap& lm, float* sc,
                                            StageA& sa, const CandRing& cr, MaskWords& mw) {
  // chunk and element indices are 32-bit (scape_create: N < 2^31), so that every address is ONE
  // IMAD.WIDE.U32 off a kernel-parameter base instead of 64-bit index arithmetic
  const uint32_t i0 = (c << 7) + ((uint32_t)lane << 2);
  // Issue order matters for latency: the mask words first (L2-resident, short latency), then the
  // 2R+1 streaming loads, and only then the gather of m_{t-1}, whose addresses depend on the
  // mask words -- it is in flight together with the streaming loads instead of after them.
  if (!DENSE) load_mask_words<PF < 2, MSPARSE && PF < 1>(p, c, lm, mw);      // whatever was not fetched ahead
  const uint32_t cw = mw.cw, pw = mw.pw;

  float th[4], mo[4], gg[R][4], ee[R][4];
  load4_f32<GUARD>(p.theta, i0, p.N, th);
  if (!MSPARSE) load4_f32<false>(p.m, i0, p.N, mo);         // own arrays are padded to Npad
#pragma unroll
  for (int r = 0; r < R; ++r) {
    load4_grad<G, GUARD>(p.g[r], i0, p.N, gg[r]);
    load4_f32<false>(p.e + r * p.e_stride, i0, p.N, ee[r]);
  }

  if constexpr (DENSE) {
    dense_compute<R, GUARD, CLIPT>(p, i0, th, mo, gg, ee, sa);
  } else {
    uint32_t mybits, jbase;
    const uint2 crk = mw.crk;
    lane_decode(cw, crk, lm, mybits, jbase);
    if (MSPARSE) {
      uint32_t pbits, pbase;
      lane_decode(pw, mw.prk, lm, pbits, pbase);
      gather_prev_m(p.pm_prev, pbits, pbase, mo);
    }
    if (PF > 0 && c_next != 0xFFFFFFFFu) load_mask_words<PF >= 2, MSPARSE && PF >= 1>(p, c_next, lm, mw);
    sparse_compute<R, GUARD, true, CLIPT, RING, kChunk>(p, c, lane, lm, i0, mybits, jbase, crk.x, crk.y >> 24, sc, sc + kChunk,
                                                        th, mo, gg, ee, sa, cr);
  }
}

// Dynamic shared memory of the register-staged kernel (sparse variants): per warp the scratch of the
// on-mask arithmetic ((R + 1) x 128 floats) and the candidate ring, then the 8 ring heads.
__host__ __device__ constexpr uint32_t step_scratch_bytes(int R) { return (uint32_t)(R + 1) * kChunk * 4u; }
__host__ __device__ constexpr uint32_t step_smem_bytes(int R, bool dense) {
  return dense ? 0u : 8u * (step_scratch_bytes(R) + kRing * 8u) + 8u * 4u + (4u << kFusedBits);
}

// Resident CTAs per SM of the register-staged kernel: sparse steps with one or two replicas are latency-bound
// (12-24 bytes per parameter in flight per lane), so they trade registers for a fourth CTA (measured, N = 2^28,
// R = 2, 90 %: 2.54 -> 2.29 ms).  With one replica and no deferred update the body fits 48 registers without a
// spill, i.e. a FIFTH CTA (40 of 64 warp slots): N = 2^28 kernel 1.111 -> 1.059 / 1.008 -> 0.956 / 0.908 -> 0.901 ms
// at 90 / 99 / 99.9 %, N = 2^30 4.45 -> 4.25 / 4.04 -> 3.89 ms.  Not further: six CTAs (40 registers) spill 68 bytes
// and lose (1.186 / 1.064 ms); R = 2 spills 44 bytes at five CTAs (1.540 -> 1.639 ms at 90 %); the deferred-update
// (CLIPT) instantiations of R = 1 gain nothing at five (8 bytes of spills; workers mode 1.094 -> 1.097 ms); three CTAs (69 registers)
// lose at R = 1 (1.223 / 1.107 ms) and at R = 2 (1.579 / 1.450 against 1.540 / 1.392).
__host__ __device__ constexpr int step_ctas_per_sm(int R, bool dense, bool clipt) {
  return dense ? (R <= 4 ? 3 : 2) : (R == 1 && !clipt) ? 5 : R <= 2 ? 4 : R <= 4 ? 3 : 2;
}
template <typename G, int R, bool DENSE, bool MSPARSE, bool CLIPT>
__global__ void __launch_bounds__(256, step_ctas_per_sm(R, DENSE, CLIPT)) scape_fused_step_kernel(const __grid_constant__ StepParams p) {
  extern __shared__ __align__(16) unsigned char step_smem[];
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
  const uint32_t wpb = blockDim.x >> 5;
  const uint32_t warp = blockIdx.x * wpb + wib;
  const uint32_t nwarps = gridDim.x * wpb;
  const uint32_t full_all = (uint32_t)(p.N >> 7);
  const uint32_t first = p.c_begin, full = p.c_end < full_all ? p.c_end : full_all;     // full chunks of this launch: [first, full)
  const LaneMap lm = lane_map(lane);
  float* sc = reinterpret_cast<float*>(step_smem + (size_t)wib * step_scratch_bytes(R));
  CandRing cr{};
  StageA sa{};
  sa.layer = kNoLayer;
  if (!DENSE) {
    cr.ring = reinterpret_cast<unsigned long long*>(step_smem + 8u * step_scratch_bytes(R)) + (size_t)wib * kRing;
    cr.head = reinterpret_cast<uint32_t*>(step_smem + 8u * (step_scratch_bytes(R) + kRing * 8u)) + wib;
    if (lane == 0) *cr.head = 0u;
    __syncwarp();
    sa.lo = p.ctl->br.lo_key; sa.hi = p.ctl->br.hi_key;
    const int hs = p.fused_hist != nullptr && p.chunk_layer == nullptr ? fused_hist_shift(sa.lo, sa.hi) : -1;
    if (hs >= 0) {                                            // CTA-uniform
      cr.hist = reinterpret_cast<uint32_t*>(step_smem + 8u * (step_scratch_bytes(R) + kRing * 8u) + 32u);
      cr.hist_shift = (uint32_t)hs;
      for (int b = threadIdx.x; b < (1 << kFusedBits); b += blockDim.x) cr.hist[b] = 0u;
      __syncthreads();
    }
    sa.seg = p.cand + (size_t)(p.seg_base + warp) * p.seg_cap;
  }
  // this warp's chunks: first + warp, + nwarps, ... (full chunks), then possibly the ragged last one
  const bool tail = (int64_t)full < p.n_chunks && (int64_t)p.c_end == p.n_chunks && warp == (full - first) % nwarps;
  MaskWords mw{};
  constexpr int PF = DENSE ? 0 : step_prefetch(R);
  if (PF > 0 && (first + warp < full || tail)) load_mask_words<PF >= 2, MSPARSE && PF >= 1>(p, first + warp < full ? first + warp : full, lm, mw);
  // (c < full before c += nwarps wraps: full + nwarps < 2^25)
  for (uint32_t c = first + warp; c < full; c += nwarps) {
    uint32_t cn = 0xFFFFFFFFu;
    if constexpr (PF > 0) cn = c + nwarps < full ? c + nwarps : tail ? full : 0xFFFFFFFFu;
    fused_chunk<G, R, DENSE, MSPARSE, false, CLIPT, true, PF>(p, c, cn, lane, lm, sc, sa, cr, mw);
  }
  if (tail) fused_chunk<G, R, DENSE, MSPARSE, true, CLIPT, true, PF>(p, full, 0xFFFFFFFFu, lane, lm, sc, sa, cr, mw);
  if (!DENSE) {
    const uint32_t n_cand = ring_drain(p, sa, cr, lane);
    if (p.chunk_layer != nullptr) warp_flush_layer(p, sa, lane);      // per-layer counts; seg_above stays 0
    uint32_t na = sa.n_above;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) na += __shfl_xor_sync(0xFFFFFFFFu, na, o);
    if (lane == 0) { p.seg_count[p.seg_base + warp] = n_cand; p.seg_above[p.seg_base + warp] = na; }
    if (cr.hist != nullptr) {                                 // the CTA's first-digit histogram joins the global one
      __syncthreads();
      for (int b = threadIdx.x; b < (1 << kFusedBits); b += blockDim.x) if (cr.hist[b]) atomicAdd(&p.fused_hist[b], cr.hist[b]);
    }
  }
  if (CLIPT && p.clip == 1) warp_store_sumsq(p, sa, warp, lane);
}


// ------------------------------------------------------------------------------------------
// Steady-state variant with shared-memory staging (sparse mask in, m stored sparsely).
//
// The LDG kernel above keeps every byte in flight in registers (2R+1 128-bit loads per lane), so
// registers bound the memory-level parallelism.  Here one producer lane per CTA streams whole tiles
// of 1024 parameters (theta, e^r, g^r slices: 1+2R bulk copies, `cp.async.bulk` = SASS UBLKCP.S.G,
// completion counted in bytes on the stage's "full" mbarrier) into a ring of shared-memory stages.
// Protocol of one stage, in order:
//   producer   waits on empty[s] (count 1), arms full[s] with the tile's byte count, issues the copies
//   consumers  (8 warps, one chunk each) wait on full[s], pull their 128-bit slices into registers,
//              compute, write theta' and e'^r back INTO the stage (in place), fence.proxy.async,
//              and meet at named barrier 1 (256 threads)
//   thread 0   sends the tile out as 1+R whole-tile bulk stores (UBLKCP.G.S), commits the group and
//              waits with cp.async.bulk.wait_group.read 1 -- i.e. until the stores of the PREVIOUS
//              tile have finished reading their stage -- and only then arrives on that previous
//              stage's empty barrier, which hands it back to the producer
// So a stage is reusable one tile after its consumers are done with it, the stores of tile i overlap
// the compute of tile i+1, and the bytes in flight are (stages - 1) x tile per CTA, independent of
// register pressure.  The scratch of the on-mask arithmetic is the warp's own theta slice (m_old)
// and e^r slices (m~^r) of the stage (their contents are in registers by then and are written back after
// sparse_compute).
// ------------------------------------------------------------------------------------------
constexpr int kTmaConsumerWarps = 8;
constexpr int kTmaTile = kTmaConsumerWarps * kChunk;          // 1024 parameters
constexpr int kTmaThreads = (kTmaConsumerWarps + 1) * 32;     // + 1 producer warp
constexpr int kTmaMaxStages = 8;
constexpr int kTmaBarrierBytes = 128;                         // flat kernel: full[8] + empty[8]
constexpr int kTmagBarrierBytes = 256;                        // grouped kernel: + mfull[2]
// Mask words by bulk copy: a CTA takes GROUPS of kTmaGroup consecutive tiles, and the producer fetches a
// group's mask words and table entries of both masks as six bulk copies (512-byte bursts of bits) into
// one of two small shared-memory buffers, one group ahead.  The consumers no longer load mask words
// from global memory at all: those loads were 5 single-sector DRAM reads per tile and mask between
// the streams' 4 KB bursts (see "small reads" in DESIGN.md §5.1) and six registers of prefetch state.
constexpr int kTmaGroup = 4;
constexpr uint32_t kMbBits = kTmaGroup * 128u;                // bytes of one mask's bits for a group (32 words per tile)
template <bool RKVIEW> __host__ __device__ constexpr uint32_t tma_mb_tab() { return kTmaGroup * (RKVIEW ? 64u : 32u); }   // rk: 8 x uint2, pre: 8 x u32 per tile
template <bool RKVIEW> __host__ __device__ constexpr uint32_t tma_mb_bytes() { return 2u * kMbBits + 2u * tma_mb_tab<RKVIEW>() + (RKVIEW ? 0u : 2u * 16u); }

template <typename G, int R>
__host__ __device__ constexpr uint32_t tma_tile_bytes() { return kTmaTile * 4u * (1u + R) + kTmaTile * (uint32_t)sizeof(G) * R; }

// Shared memory one SM offers the staged kernel: two resident CTAs, each with its barriers and 1 KB that the
// driver reserves per CTA.  The kernel is only worth launching with at least 3 stages per CTA and 2 CTAs
// per SM (measured: one CTA of 8 consumer warps per SM cannot keep up with HBM, 4.8 vs 5.95 TB/s).
constexpr uint32_t kSmemPerSm = 227u * 1024u;
template <typename G, int R>
__host__ __device__ constexpr int tma_stages_two_ctas() { return (int)((kSmemPerSm / 2u - 1024u - kTmaBarrierBytes) / tma_tile_bytes<G, R>()); }
template <typename G, int R>
__host__ __device__ constexpr int tmag_stages_two_ctas() {
  return (int)((kSmemPerSm / 2u - 1024u - kTmagBarrierBytes - 2u * tma_mb_bytes<true>()) / tma_tile_bytes<G, R>());
}
template <typename G, int R>
__host__ __device__ constexpr bool tma_can_launch() { return tma_stages_two_ctas<G, R>() >= 3 && tmag_stages_two_ctas<G, R>() >= 3; }

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "WAIT_%=:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra DONE_%=;\n\t"
      "bra WAIT_%=;\n\t"
      "DONE_%=:\n\t}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// 1-D bulk copy global -> shared, completion signalled on `bar` in bytes; L2 evict-first policy
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src, uint32_t bytes, uint64_t* bar, uint64_t policy) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
               ::"r"(smem_u32(dst_smem)), "l"(src), "r"(bytes), "r"(smem_u32(bar)), "l"(policy) : "memory");
}

// own word of bits of the current / previous mask + their table entries: (c0, c1) / (p0, p1) = rk[c] when
// RKVIEW, else {pre[8T + lane % 8], trank[T]}.  RKVIEW is the instantiation for per-layer refresh: evenly
// spread masks make the consumer warps, not HBM, the bound there, and rk decodes in fewer instructions.
struct TmaMaskWords { uint32_t cw, pw, c0, c1, p0, p1; };
struct TmaTileState { uint32_t mybits, jbase, r0, cnt; float mo[4]; };

// this lane's mask words of chunk `warp` of tile t (0 .. kTmaGroup-1) of the group held in buffer mb
template <bool RKVIEW>
__device__ __forceinline__ void tma_read_words(const unsigned char* mb, int t, int warp, const LaneMap& lm, TmaMaskWords& w) {
  const uint32_t* cb = reinterpret_cast<const uint32_t*>(mb);
  const uint32_t* pb = reinterpret_cast<const uint32_t*>(mb + kMbBits);
  w.cw = cb[t * 32 + warp * 4 + lm.ws];
  w.pw = pb[t * 32 + warp * 4 + lm.ws];
  const unsigned char* ct = mb + 2u * kMbBits;
  const unsigned char* pt = ct + tma_mb_tab<RKVIEW>();
  if constexpr (RKVIEW) {
    const uint2 a = reinterpret_cast<const uint2*>(ct)[t * 8 + warp], b = reinterpret_cast<const uint2*>(pt)[t * 8 + warp];
    w.c0 = a.x; w.c1 = a.y; w.p0 = b.x; w.p1 = b.y;
  } else {
    const uint32_t li = (uint32_t)t * 8u + (lm.sh >> 2);      // (lm.sh >> 2 = lane % 8)
    const uint32_t* tr = reinterpret_cast<const uint32_t*>(pt + tma_mb_tab<RKVIEW>());
    w.c0 = reinterpret_cast<const uint32_t*>(ct)[li]; w.c1 = tr[t];
    w.p0 = reinterpret_cast<const uint32_t*>(pt)[li]; w.p1 = tr[4 + t];
  }
}
template <bool RKVIEW>
__device__ __forceinline__ void tma_load_words(const StepParams& p, uint32_t c, const LaneMap& lm, TmaMaskWords& w) {
  w.cw = __ldg(p.cur_bits + (c << 2) + lm.ws);
  w.pw = __ldg(p.prev_bits + (c << 2) + lm.ws);
  if constexpr (RKVIEW) {
    const uint2 a = __ldg(p.cur_rk + c), b = __ldg(p.prev_rk + c);
    w.c0 = a.x; w.c1 = a.y; w.p0 = b.x; w.p1 = b.y;
  } else {
    const uint32_t pi = (c & ~7u) + (lm.sh >> 2);             // (lm.sh >> 2 = lane % 8)
    w.c0 = __ldg(p.cur_pre + pi); w.c1 = __ldg(p.cur_trank + (c >> 3));
    w.p0 = __ldg(p.prev_pre + pi); w.p1 = __ldg(p.prev_trank + (c >> 3));
  }
}
// decode a chunk's mask words for this lane and start the gather of m_{t-1}
template <bool RKVIEW>
__device__ __forceinline__ void tma_decode_gather(const StepParams& p, const TmaMaskWords& w, const LaneMap& lm, uint32_t pos, TmaTileState& st) {
  uint32_t pbits, pbase;
  const int lane = (int)(lm.ws * 8u + (lm.sh >> 2));
  const uint2 crk = RKVIEW ? make_uint2(w.c0, w.c1) : chunk_rank(w.c0, w.c1, pos, lane);
  const uint2 prk = RKVIEW ? make_uint2(w.p0, w.p1) : chunk_rank(w.p0, w.p1, pos, lane);
  lane_decode(w.cw, crk, lm, st.mybits, st.jbase);
  st.r0 = crk.x; st.cnt = crk.y >> 24;
  lane_decode(w.pw, prk, lm, pbits, pbase);
  gather_prev_m(p.pm_prev, pbits, pbase, st.mo);
}

// 1-D bulk copy shared -> global (whole-tile store), tracked by the thread's bulk async-group
__device__ __forceinline__ void bulk_s2g(void* dst, const void* src_smem, uint32_t bytes, uint64_t policy) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group.L2::cache_hint [%0], [%1], %2, %3;"
               ::"l"(dst), "r"(smem_u32(src_smem)), "r"(bytes), "l"(policy) : "memory");
}

// The tiles of one CTA: groups g = blockIdx.x, + gridDim.x, ... of kTmaGroup consecutive tiles (the last group
// of the shard may be short); j = ordinal of the group within this CTA (its mask buffer is j & 1).
struct TmaPos { int64_t g; int t; int j; };
__device__ __forceinline__ bool tma_pos_valid(const TmaPos& q, int64_t n_tiles) { return q.g * kTmaGroup + q.t < n_tiles; }
__device__ __forceinline__ TmaPos tma_pos_next(const TmaPos& q, int64_t n_tiles) {
  TmaPos n = q;
  if (++n.t == kTmaGroup || n.g * kTmaGroup + n.t >= n_tiles) { n.t = 0; n.g += gridDim.x; n.j += 1; }
  return n;
}

// One tile of one consumer warp: read the next tile's mask words from the group's buffer and start its
// gather of m, wait for this tile's bytes, pull them out of shared memory, compute, write the results back
// into the stage; thread 0 then issues the tile's bulk stores and releases the previous stage (protocol above).
template <typename G, int R, bool CLIPT, bool RKVIEW>
__device__ __forceinline__ void tmag_consume_tile(const StepParams& p, const TmaPos& pos, int64_t n_tiles, bool first,
                                                 int warp, int lane, const LaneMap& lm, unsigned char* stage0, const unsigned char* mb0,
                                                 uint64_t* full, uint64_t* empty, uint64_t* mfull,
                                                 int& s, uint32_t& ph, int n_stages,
                                                 TmaTileState& cur, TmaTileState& nxt, StageA& sa) {
  constexpr uint32_t TILE = tma_tile_bytes<G, R>();
  constexpr uint32_t OFF_E = kTmaTile * 4u, OFF_G = kTmaTile * 4u * (1u + R);
  const int64_t tile = pos.g * kTmaGroup + pos.t;
  const uint32_t c = (uint32_t)tile * kTmaConsumerWarps + warp;
  const uint32_t i0 = (c << 7) + ((uint32_t)lane << 2);
  {
    const TmaPos nx = tma_pos_next(pos, n_tiles);
    if (tma_pos_valid(nx, n_tiles)) {
      if (nx.t == 0) mbar_wait(&mfull[nx.j & 1], (uint32_t)(nx.j >> 1) & 1u);      // the next group's mask words have landed
      TmaMaskWords nw;
      tma_read_words<RKVIEW>(mb0 + (size_t)(nx.j & 1) * tma_mb_bytes<RKVIEW>(), nx.t, warp, lm, nw);
      tma_decode_gather<RKVIEW>(p, nw, lm, (uint32_t)warp, nxt);
    }
  }
  mbar_wait(&full[s], ph);
  const unsigned char* base = stage0 + (size_t)s * TILE;
  const uint32_t off = (uint32_t)(warp * kChunk + (lane << 2));
  float th[4], gg[R][4], ee[R][4];
  {
    const float4 t = *reinterpret_cast<const float4*>(base + off * 4u);
    th[0] = t.x; th[1] = t.y; th[2] = t.z; th[3] = t.w;
  }
#pragma unroll
  for (int r = 0; r < R; ++r) {
    const float4 t = *reinterpret_cast<const float4*>(base + OFF_E + r * (kTmaTile * 4u) + off * 4u);
    ee[r][0] = t.x; ee[r][1] = t.y; ee[r][2] = t.z; ee[r][3] = t.w;
    if constexpr (sizeof(G) == 4) {
      const float4 g = *reinterpret_cast<const float4*>(base + OFF_G + r * (kTmaTile * 4u) + off * 4u);
      gg[r][0] = g.x; gg[r][1] = g.y; gg[r][2] = g.z; gg[r][3] = g.w;
    } else {
      const uint2 g = *reinterpret_cast<const uint2*>(base + OFF_G + r * (kTmaTile * 2u) + off * 2u);
      gg[r][0] = __uint_as_float(g.x << 16); gg[r][1] = __uint_as_float(g.x & 0xFFFF0000u);
      gg[r][2] = __uint_as_float(g.y << 16); gg[r][3] = __uint_as_float(g.y & 0xFFFF0000u);
    }
  }
  // Results go back into the stage (in place) and leave as whole-tile bulk stores: 4 KB bursts
  // per stream instead of 512-byte warp stores.
  // scratch of the on-mask arithmetic: this warp's own theta slice (m_old) and e^r slices (m~^r) of
  // the stage (their contents are in registers now and are written back only after sparse_compute)
  unsigned char* wbase = stage0 + (size_t)s * TILE;
  __syncwarp();
  sparse_compute<R, false, false, CLIPT, false, kTmaTile>(p, c, lane, lm, i0, cur.mybits, cur.jbase, cur.r0, cur.cnt,
                                                          reinterpret_cast<float*>(wbase) + warp * kChunk,
                                                          reinterpret_cast<float*>(wbase + OFF_E) + warp * kChunk, th, cur.mo, gg, ee, sa,
                                                          CandRing{});
  *reinterpret_cast<float4*>(wbase + off * 4u) = make_float4(th[0], th[1], th[2], th[3]);
#pragma unroll
  for (int r = 0; r < R; ++r)
    *reinterpret_cast<float4*>(wbase + OFF_E + r * (kTmaTile * 4u) + off * 4u) = make_float4(ee[r][0], ee[r][1], ee[r][2], ee[r][3]);
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  asm volatile("bar.sync 1, %0;" ::"n"(kTmaConsumerWarps * 32) : "memory");
  if (threadIdx.x == 0) {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    const int64_t e0 = tile * kTmaTile;
    bulk_s2g(p.theta + e0, wbase, kTmaTile * 4u, pol);
#pragma unroll
    for (int r = 0; r < R; ++r) bulk_s2g(p.e + r * p.e_stride + e0, wbase + OFF_E + r * (kTmaTile * 4u), kTmaTile * 4u, pol);
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    // the stores of the PREVIOUS tile have finished reading their stage: hand it back
    asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory");
    if (!first) mbar_arrive(&empty[s == 0 ? n_stages - 1 : s - 1]);
  }
  if (++s == n_stages) { s = 0; ph ^= 1u; }
}

template <typename G, int R, bool CLIPT, bool RKVIEW>
__global__ void __launch_bounds__(kTmaThreads, 2) scape_fused_tmag_kernel(const __grid_constant__ StepParams p, int n_stages) {
  extern __shared__ __align__(128) unsigned char smem[];
  constexpr uint32_t TILE = tma_tile_bytes<G, R>();
  constexpr uint32_t OFF_E = kTmaTile * 4u, OFF_G = kTmaTile * 4u * (1u + R);
  constexpr uint32_t MB = tma_mb_bytes<RKVIEW>();
  uint64_t* full = reinterpret_cast<uint64_t*>(smem);
  uint64_t* empty = full + kTmaMaxStages;
  uint64_t* mfull = empty + kTmaMaxStages;                    // [2]: a group's mask words have landed
  unsigned char* mb0 = smem + kTmagBarrierBytes;              // two mask buffers
  unsigned char* stage0 = mb0 + 2u * MB;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int64_t n_tiles = p.N / kTmaTile;                     // full tiles; the rest goes through the LDG path
  const int64_t n_groups = (n_tiles + kTmaGroup - 1) / kTmaGroup;

  if (threadIdx.x == 0) {
    for (int s = 0; s < n_stages; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], 1); }
    mbar_init(&mfull[0], 1); mbar_init(&mfull[1], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  if (warp == kTmaConsumerWarps) {
    // ===== producer: one lane streams the tiles of this CTA and, one group ahead, the groups' mask words =====
    // (Tried: the idle lanes prefetching each coming tile's range of the previous packed mean into L2,
    // so that the consumers' gather of m hits there.  The hit rate rose from 11 to 18 %, the kernel got
    // SLOWER -- 13.75 vs 13.62 ms on the headline shard, 2.43 vs 2.39 ms at N = 2^28, R = 4 -- because
    // whole-line prefetches are more small reads between the streams' bursts than the sectors the
    // gather touches.  The consumers do wait for the gather, but only while the streams are the bound.)
    if (lane == 0) {
      uint64_t policy, keep;
      asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(policy));
      asm volatile("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(keep));
      // mask words of group g -> buffer j & 1 (the table arrays are padded to whole groups: scape.cu)
      auto load_masks = [&](int64_t g, int j) {
        unsigned char* mb = mb0 + (size_t)(j & 1) * MB;
        uint64_t* bar = &mfull[j & 1];
        mbar_expect_tx(bar, MB);
        bulk_g2s(mb, p.cur_bits + g * (kMbBits / 4u), kMbBits, bar, keep);
        bulk_g2s(mb + kMbBits, p.prev_bits + g * (kMbBits / 4u), kMbBits, bar, keep);
        unsigned char* ct = mb + 2u * kMbBits;
        if constexpr (RKVIEW) {
          bulk_g2s(ct, p.cur_rk + g * (kTmaGroup * 8), tma_mb_tab<true>(), bar, keep);
          bulk_g2s(ct + tma_mb_tab<true>(), p.prev_rk + g * (kTmaGroup * 8), tma_mb_tab<true>(), bar, keep);
        } else {
          bulk_g2s(ct, p.cur_pre + g * (kTmaGroup * 8), tma_mb_tab<false>(), bar, keep);
          bulk_g2s(ct + tma_mb_tab<false>(), p.prev_pre + g * (kTmaGroup * 8), tma_mb_tab<false>(), bar, keep);
          bulk_g2s(ct + 2u * tma_mb_tab<false>(), p.cur_trank + g * kTmaGroup, 16u, bar, keep);
          bulk_g2s(ct + 2u * tma_mb_tab<false>() + 16u, p.prev_trank + g * kTmaGroup, 16u, bar, keep);
        }
      };
      int s = 0; uint32_t ph = 0;
      TmaPos q{(int64_t)blockIdx.x, 0, 0};
      if (q.g < n_groups) load_masks(q.g, 0);
      for (; tma_pos_valid(q, n_tiles); q = tma_pos_next(q, n_tiles)) {
        mbar_wait(&empty[s], ph ^ 1u);                         // every consumer warp has read the old contents
        // The buffer of group j + 1 is the one group j - 1 used: free once the LAST tile of j - 1 has been
        // released, which the wait above implies from tile n_stages - 1 of group j on (n_stages <= kTmaGroup).
        if (q.t == n_stages - 1 && q.g + gridDim.x < n_groups) load_masks(q.g + gridDim.x, q.j + 1);
        mbar_expect_tx(&full[s], TILE);
        unsigned char* base = stage0 + (size_t)s * TILE;
        const int64_t e0 = (q.g * kTmaGroup + q.t) * kTmaTile;
        bulk_g2s(base, p.theta + e0, kTmaTile * 4u, &full[s], policy);
#pragma unroll
        for (int r = 0; r < R; ++r)
          bulk_g2s(base + OFF_E + r * (kTmaTile * 4u), p.e + r * p.e_stride + e0, kTmaTile * 4u, &full[s], policy);
#pragma unroll
        for (int r = 0; r < R; ++r)
          bulk_g2s(base + OFF_G + r * (kTmaTile * (uint32_t)sizeof(G)),
                   reinterpret_cast<const unsigned char*>(p.g[r]) + e0 * (int64_t)sizeof(G),
                   kTmaTile * (uint32_t)sizeof(G), &full[s], policy);
        if (++s == n_stages) { s = 0; ph ^= 1u; }
      }
    }
    return;
  }

  // ===== consumers =====
  const LaneMap lm = lane_map(lane);
  const int64_t gwarp = (int64_t)blockIdx.x * kTmaConsumerWarps + warp;     // candidate segment of this warp
  StageA sa{};
  sa.layer = kNoLayer;
  sa.lo = p.ctl->br.lo_key; sa.hi = p.ctl->br.hi_key;
  sa.seg = p.cand + (size_t)gwarp * p.seg_cap;

  // Software pipeline of the dependent accesses: the gather of m_{t-1} (whose addresses come from the
  // previous mask's words) is issued one tile ahead; the mask words themselves arrive by bulk copy one
  // group ahead.  The per-tile state ping-pongs between two register sets (A, B).
  TmaPos q{(int64_t)blockIdx.x, 0, 0};
  TmaTileState stA{}, stB{};
  if (tma_pos_valid(q, n_tiles)) {
    mbar_wait(&mfull[0], 0u);
    TmaMaskWords w0;
    tma_read_words<RKVIEW>(mb0, 0, warp, lm, w0);
    tma_decode_gather<RKVIEW>(p, w0, lm, (uint32_t)warp, stA);
  }
  int s = 0; uint32_t ph = 0;
  bool first = true;
  while (tma_pos_valid(q, n_tiles)) {
    tmag_consume_tile<G, R, CLIPT, RKVIEW>(p, q, n_tiles, first, warp, lane, lm, stage0, mb0, full, empty, mfull, s, ph, n_stages, stA, stB, sa);
    first = false;
    q = tma_pos_next(q, n_tiles);
    if (!tma_pos_valid(q, n_tiles)) break;
    tmag_consume_tile<G, R, CLIPT, RKVIEW>(p, q, n_tiles, first, warp, lane, lm, stage0, mb0, full, empty, mfull, s, ph, n_stages, stB, stA, sa);
    q = tma_pos_next(q, n_tiles);
  }
  if (threadIdx.x == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");   // stores have landed
  asm volatile("bar.sync 1, %0;" ::"n"(kTmaConsumerWarps * 32) : "memory");          // ... and every consumer warp knows

  // chunks past the last full tile (fewer than 8, the last one possibly ragged): LDG path
  {
    const uint32_t c = (uint32_t)n_tiles * kTmaConsumerWarps + warp;
    if ((int64_t)c < p.n_chunks && blockIdx.x == (unsigned)(n_tiles % gridDim.x)) {
      // (all bulk stores of this CTA have completed: the first stage serves as scratch)
      float* sc = reinterpret_cast<float*>(stage0) + warp * ((R + 1) * kChunk);
      MaskWords mw;
      if (((int64_t)(c + 1) << 7) <= p.N) fused_chunk<G, R, false, true, false, CLIPT, false, 0>(p, c, 0xFFFFFFFFu, lane, lm, sc, sa, CandRing{}, mw);
      else fused_chunk<G, R, false, true, true, CLIPT, false, 0>(p, c, 0xFFFFFFFFu, lane, lm, sc, sa, CandRing{}, mw);
    }
  }
  if (p.chunk_layer != nullptr) warp_flush_layer(p, sa, lane);        // per-layer counts; seg_above stays 0
  uint32_t na = sa.n_above;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) na += __shfl_xor_sync(0xFFFFFFFFu, na, o);
  if (lane == 0) { p.seg_count[gwarp] = sa.cursor; p.seg_above[gwarp] = na; }
  if (CLIPT && p.clip == 1) warp_store_sumsq(p, sa, gwarp, lane);
}


// ------------------------------------------------------------------------------------------
// The flat-top-k form of the staged kernel: tiles blockIdx.x, + gridDim.x, ...; mask words loaded from global
// memory two tiles ahead by the consumer warps; one more stage fits.  HBM-bound there (0.97 of the measured
// peak), and measured ahead of the grouped form above on flat masks (13.67 vs 13.93 ms on the headline
// shard), while the grouped form wins where the consumer warps are the bound (per-layer refresh: 13.97
// vs 14.6 ms) -- see DESIGN.md §5.1.
// ------------------------------------------------------------------------------------------
// One tile of one consumer warp: start the next tile's gather of m, wait for this tile's bytes, pull
// them out of shared memory, compute, write the results back into the stage; thread 0 then issues
// the tile's bulk stores and releases the previous stage (protocol above).
template <typename G, int R, bool CLIPT, bool RKVIEW>
__device__ __forceinline__ void tma_consume_tile(const StepParams& p, int64_t tile, int64_t n_tiles, int64_t tstride,
                                                 int warp, int lane, const LaneMap& lm, unsigned char* stage0, uint64_t* full, uint64_t* empty,
                                                 int& s, uint32_t& ph, int n_stages, TmaMaskWords& nw,
                                                 TmaTileState& cur, TmaTileState& nxt, StageA& sa) {
  constexpr uint32_t TILE = tma_tile_bytes<G, R>();
  constexpr uint32_t OFF_E = kTmaTile * 4u, OFF_G = kTmaTile * 4u * (1u + R);
  const uint32_t c = (uint32_t)tile * kTmaConsumerWarps + warp;
  const uint32_t i0 = (c << 7) + ((uint32_t)lane << 2);
  if (tile + tstride < n_tiles) {
    tma_decode_gather<RKVIEW>(p, nw, lm, (uint32_t)warp, nxt);
    if (tile + 2 * tstride < n_tiles) tma_load_words<RKVIEW>(p, (uint32_t)(tile + 2 * tstride) * kTmaConsumerWarps + warp, lm, nw);
  }
  mbar_wait(&full[s], ph);
  const unsigned char* base = stage0 + (size_t)s * TILE;
  const uint32_t off = (uint32_t)(warp * kChunk + (lane << 2));
  float th[4], gg[R][4], ee[R][4];
  {
    const float4 t = *reinterpret_cast<const float4*>(base + off * 4u);
    th[0] = t.x; th[1] = t.y; th[2] = t.z; th[3] = t.w;
  }
#pragma unroll
  for (int r = 0; r < R; ++r) {
    const float4 t = *reinterpret_cast<const float4*>(base + OFF_E + r * (kTmaTile * 4u) + off * 4u);
    ee[r][0] = t.x; ee[r][1] = t.y; ee[r][2] = t.z; ee[r][3] = t.w;
    if constexpr (sizeof(G) == 4) {
      const float4 g = *reinterpret_cast<const float4*>(base + OFF_G + r * (kTmaTile * 4u) + off * 4u);
      gg[r][0] = g.x; gg[r][1] = g.y; gg[r][2] = g.z; gg[r][3] = g.w;
    } else {
      const uint2 g = *reinterpret_cast<const uint2*>(base + OFF_G + r * (kTmaTile * 2u) + off * 2u);
      gg[r][0] = __uint_as_float(g.x << 16); gg[r][1] = __uint_as_float(g.x & 0xFFFF0000u);
      gg[r][2] = __uint_as_float(g.y << 16); gg[r][3] = __uint_as_float(g.y & 0xFFFF0000u);
    }
  }
  // Results go back into the stage (in place) and leave as whole-tile bulk stores: 4 KB bursts
  // per stream instead of 512-byte warp stores.
  // scratch of the on-mask arithmetic: this warp's own theta slice (m_old) and e^r slices (m~^r) of
  // the stage (their contents are in registers now and are written back only after sparse_compute)
  unsigned char* wbase = stage0 + (size_t)s * TILE;
  __syncwarp();
  sparse_compute<R, false, false, CLIPT, false, kTmaTile>(p, c, lane, lm, i0, cur.mybits, cur.jbase, cur.r0, cur.cnt,
                                                          reinterpret_cast<float*>(wbase) + warp * kChunk,
                                                          reinterpret_cast<float*>(wbase + OFF_E) + warp * kChunk, th, cur.mo, gg, ee, sa,
                                                          CandRing{});
  *reinterpret_cast<float4*>(wbase + off * 4u) = make_float4(th[0], th[1], th[2], th[3]);
#pragma unroll
  for (int r = 0; r < R; ++r)
    *reinterpret_cast<float4*>(wbase + OFF_E + r * (kTmaTile * 4u) + off * 4u) = make_float4(ee[r][0], ee[r][1], ee[r][2], ee[r][3]);
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  asm volatile("bar.sync 1, %0;" ::"n"(kTmaConsumerWarps * 32) : "memory");
  if (threadIdx.x == 0) {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    const int64_t e0 = tile * kTmaTile;
    bulk_s2g(p.theta + e0, wbase, kTmaTile * 4u, pol);
#pragma unroll
    for (int r = 0; r < R; ++r) bulk_s2g(p.e + r * p.e_stride + e0, wbase + OFF_E + r * (kTmaTile * 4u), kTmaTile * 4u, pol);
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    // the stores of the PREVIOUS tile have finished reading their stage: hand it back
    asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory");
    if (tile - tstride >= (int64_t)(p.c_begin >> 3)) mbar_arrive(&empty[s == 0 ? n_stages - 1 : s - 1]);       // (not after this CTA's first tile)
  }
  if (++s == n_stages) { s = 0; ph ^= 1u; }
}

template <typename G, int R, bool CLIPT, bool RKVIEW>
__global__ void __launch_bounds__(kTmaThreads, 2) scape_fused_tma_kernel(const __grid_constant__ StepParams p, int n_stages) {
  extern __shared__ __align__(128) unsigned char smem[];
  constexpr uint32_t TILE = tma_tile_bytes<G, R>();
  constexpr uint32_t OFF_E = kTmaTile * 4u, OFF_G = kTmaTile * 4u * (1u + R);
  uint64_t* full = reinterpret_cast<uint64_t*>(smem);
  uint64_t* empty = full + kTmaMaxStages;
  unsigned char* stage0 = smem + kTmaBarrierBytes;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int64_t t_first = p.c_begin >> 3;                     // this launch: tiles [t_first, n_tiles)
  const int64_t n_tiles = min((int64_t)(p.N / kTmaTile), (int64_t)(p.c_end >> 3));   // full tiles; the rest goes through the LDG path

  if (threadIdx.x == 0) {
    for (int s = 0; s < n_stages; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], 1); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  if (warp == kTmaConsumerWarps) {
    // ===== producer: one lane streams the tiles of this CTA =====
    // (Tried: the idle lanes prefetching each coming tile's range of the previous packed mean into L2,
    // so that the consumers' gather of m hits there.  The hit rate rose from 11 to 18 %, the kernel got
    // SLOWER -- 13.75 vs 13.62 ms on the headline shard, 2.43 vs 2.39 ms at N = 2^28, R = 4 -- because
    // whole-line prefetches are more small reads between the streams' bursts than the sectors the
    // gather touches.  The consumers do wait for the gather, but only while the streams are the bound.)
    if (lane == 0) {
      uint64_t policy;
      asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(policy));
      int s = 0; uint32_t ph = 0;
      for (int64_t tile = t_first + blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        mbar_wait(&empty[s], ph ^ 1u);                         // every consumer warp has read the old contents
        mbar_expect_tx(&full[s], TILE);
        unsigned char* base = stage0 + (size_t)s * TILE;
        const int64_t e0 = tile * kTmaTile;
        bulk_g2s(base, p.theta + e0, kTmaTile * 4u, &full[s], policy);
#pragma unroll
        for (int r = 0; r < R; ++r)
          bulk_g2s(base + OFF_E + r * (kTmaTile * 4u), p.e + r * p.e_stride + e0, kTmaTile * 4u, &full[s], policy);
#pragma unroll
        for (int r = 0; r < R; ++r)
          bulk_g2s(base + OFF_G + r * (kTmaTile * (uint32_t)sizeof(G)),
                   reinterpret_cast<const unsigned char*>(p.g[r]) + e0 * (int64_t)sizeof(G),
                   kTmaTile * (uint32_t)sizeof(G), &full[s], policy);
        if (++s == n_stages) { s = 0; ph ^= 1u; }
      }
    }
    return;
  }

  // ===== consumers =====
  const LaneMap lm = lane_map(lane);
  const int64_t gwarp = (int64_t)p.seg_base + (int64_t)blockIdx.x * kTmaConsumerWarps + warp;     // candidate segment of this warp
  StageA sa{};
  sa.layer = kNoLayer;
  sa.lo = p.ctl->br.lo_key; sa.hi = p.ctl->br.hi_key;
  sa.seg = p.cand + (size_t)gwarp * p.seg_cap;

  // Software pipeline of the small dependent accesses, so that none of their latency is exposed
  // once a tile has landed: mask words are fetched two tiles ahead, and the gather of m_{t-1}
  // (whose addresses come from the previous mask's words) one tile ahead.  The per-tile state
  // ping-pongs between two register sets (A, B) so that no register move has to wait for a load.
  const int64_t tstride = gridDim.x;
  int64_t tile = t_first + blockIdx.x;
  TmaMaskWords nw{};                                   // raw words of the NEXT tile
  TmaTileState stA{}, stB{};
  if (tile < n_tiles) {
    TmaMaskWords w0;
    tma_load_words<RKVIEW>(p, (uint32_t)tile * kTmaConsumerWarps + warp, lm, w0);
    if (tile + tstride < n_tiles) tma_load_words<RKVIEW>(p, (uint32_t)(tile + tstride) * kTmaConsumerWarps + warp, lm, nw);
    tma_decode_gather<RKVIEW>(p, w0, lm, (uint32_t)warp, stA);
  }
  int s = 0; uint32_t ph = 0;
  while (tile < n_tiles) {
    tma_consume_tile<G, R, CLIPT, RKVIEW>(p, tile, n_tiles, tstride, warp, lane, lm, stage0, full, empty, s, ph, n_stages, nw, stA, stB, sa);
    tile += tstride;
    if (tile >= n_tiles) break;
    tma_consume_tile<G, R, CLIPT, RKVIEW>(p, tile, n_tiles, tstride, warp, lane, lm, stage0, full, empty, s, ph, n_stages, nw, stB, stA, sa);
    tile += tstride;
  }
  if (threadIdx.x == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");   // stores have landed
  asm volatile("bar.sync 1, %0;" ::"n"(kTmaConsumerWarps * 32) : "memory");          // ... and every consumer warp knows

  // chunks past the last full tile (fewer than 8, the last one possibly ragged): LDG path
  {
    const uint32_t c = (uint32_t)n_tiles * kTmaConsumerWarps + warp;
    if ((int64_t)c < p.n_chunks && (int64_t)p.c_end == p.n_chunks && blockIdx.x == (unsigned)((n_tiles - t_first) % gridDim.x)) {
      // (all bulk stores of this CTA have completed: the first stage serves as scratch)
      float* sc = reinterpret_cast<float*>(stage0) + warp * ((R + 1) * kChunk);
      MaskWords mw;
      if (((int64_t)(c + 1) << 7) <= p.N) fused_chunk<G, R, false, true, false, CLIPT, false, 0>(p, c, 0xFFFFFFFFu, lane, lm, sc, sa, CandRing{}, mw);
      else fused_chunk<G, R, false, true, true, CLIPT, false, 0>(p, c, 0xFFFFFFFFu, lane, lm, sc, sa, CandRing{}, mw);
    }
  }
  if (p.chunk_layer != nullptr) warp_flush_layer(p, sa, lane);        // per-layer counts; seg_above stays 0
  uint32_t na = sa.n_above;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) na += __shfl_xor_sync(0xFFFFFFFFu, na, o);
  if (lane == 0) { p.seg_count[gwarp] = sa.cursor; p.seg_above[gwarp] = na; }
  if (CLIPT && p.clip == 1) warp_store_sumsq(p, sa, gwarp, lane);
}


}  // namespace scapek
