// scape_kernels.cuh — sm_100a kernels of the SCAPE step (Algorithm 1, :131-174).
//
// Data layout: the shard is cut into CHUNKS of 128 consecutive
// parameters; one warp handles one chunk per loop trip, lane l owning elements 4l..4l+3
// (one 128-bit access per fp32 array, one 64-bit access per bf16 array).  A mask is stored as
// bits (word i/32, bit i%32 => one uint4 per chunk) plus `rank128[c]`, the number of set bits
// before chunk c, so the packed position of a selected element is rank128[c] + popc(bits
// before it inside the chunk): the pack of Alg. 1 l.9 needs no atomics and keeps ascending
// index order.
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
  unsigned int pad1;
  unsigned long long base;    // fast route: the radix passes run on K64 - base (base = lo_key << 32), see sel_decide_kernel
  Bracket br;                 // predicted bracket for the COMING step's fused pass
  unsigned long long cand_cap_total;   // n_seg * seg_cap of the last fused pass
  int hit;                    // this step: 1 = the bracket held (candidate list), 0 = general path
  unsigned long long n_fast, n_general;   // statistics (scape_select_stats)
  unsigned long long n_above, n_cand;     // this step's counts from the fused pass
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
};

struct StepParams {
  float* theta;                 // [N] caller-owned
  float* m;                     // [Npad]
  float* e;                     // [R][e_stride]
  int64_t e_stride;
  const void* g[kMaxR];         // R caller-owned gradient buffers
  const uint32_t* cur_bits;     // [Npad/32]   (unused when DENSE)
  const uint32_t* cur_rank;     // [Npad/128]
  float* packed;                // [R][packed_stride] or nullptr (DENSE without keep_dense_pack)
  int64_t packed_stride;
  float* packed_mean;           // [k] b- of this step = m_t in packed form (unused when DENSE)
  // m_{t-1} stored sparsely (MSPARSE): it is zero off the mask the previous step used (Eq. 4,
  // PAPER.md:197), so it lives as that step's packed mean, addressed through that mask
  const uint32_t* prev_bits;    // [Npad/32]
  const uint32_t* prev_rank;    // [Npad/128]
  const float* pm_prev;         // [k]
  int64_t N;
  int64_t n_chunks;             // ceil(N/128)
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
  uint32_t compact_min;         // selected entries per chunk from which l.10-16 run in compacted form
  // stage 2 fused into the pass (sparse variant only)
  const SelState* ctl;          // bracket predicted by the previous step
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
__device__ __forceinline__ void load4_f32(const float* __restrict__ p, int64_t i0, int64_t N, float (&v)[4]) {
  if (!GUARD) {
    const float4 t = __ldcs(reinterpret_cast<const float4*>(p + i0));
    v[0] = t.x; v[1] = t.y; v[2] = t.z; v[3] = t.w;
  } else {
#pragma unroll
    for (int q = 0; q < 4; ++q) v[q] = (i0 + q < N) ? __ldcs(p + i0 + q) : 0.0f;
  }
}

template <bool GUARD>
__device__ __forceinline__ void store4_f32(float* __restrict__ p, int64_t i0, int64_t N, const float (&v)[4]) {
  if (!GUARD) {
    __stcs(reinterpret_cast<float4*>(p + i0), make_float4(v[0], v[1], v[2], v[3]));
  } else {
#pragma unroll
    for (int q = 0; q < 4; ++q) if (i0 + q < N) __stcs(p + i0 + q, v[q]);
  }
}

// Gradient loads: fp32, or bf16 widened exactly (S16) by placing the 16 bits in the high half.
template <typename G, bool GUARD>
__device__ __forceinline__ void load4_grad(const void* __restrict__ base, int64_t i0, int64_t N, float (&v)[4]) {
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

__device__ __forceinline__ void lane_mask_bits(const uint32_t* __restrict__ bits, const uint32_t* __restrict__ rank,
                                               int64_t c, int lane, uint32_t& mybits, uint32_t& jbase) {
  const uint4 mw = __ldg(reinterpret_cast<const uint4*>(bits) + c);
  lane_bits_from_words(mw, __ldg(rank + c), lane, mybits, jbase);
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
//
// Sparse steps: the selected entries of a chunk (cnt of 128; ~13 at 90 % sparsity, ~1 at 99 %) are
// scattered over the lanes, so running l.10-16 (IEEE divisions, square root) where they sit would
// mean four divergent passes with a few active lanes each.  Instead every lane parks (sum_r m~^r,
// m_old) of its selected entries in a warp-private scratch at the entry's rank inside the chunk,
// and lane l then runs l.10-16 for the entry of rank l: one pass, consecutive lanes, b- stored
// coalesced.  The update u comes back through the same scratch.
//   r0 = rank128[c]; cnt = set bits of the chunk; scs, scm = 128 floats each, private to this warp
template <int R, bool DENSE, bool GUARD, bool STORE = true, bool CLIPT = true, bool COMPACT = true>
__device__ __forceinline__ void fused_compute(const StepParams& p, int64_t c, int lane, int64_t i0,
                                              uint32_t mybits, uint32_t jbase, uint32_t r0, uint32_t cnt, float* scs, float* scm,
                                              float (&th)[4], const float (&mo)[4],
                                              float (&gg)[R][4], float (&ee)[R][4], StageA& sa) {
  uint32_t key0[4];             // bits(|m~^0|): the selection statistic of l.11
  if constexpr (DENSE) {
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
      key0[q] = __float_as_uint(mt[0]) & 0x7FFFFFFFu;
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
      if (CLIPT && p.clip) {
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
    if (STORE) {
      store4_f32<GUARD>(p.theta, i0, p.N, th);
#pragma unroll
      for (int r = 0; r < R; ++r) store4_f32<false>(p.e + r * p.e_stride, i0, p.N, ee[r]);
    }
    store4_f32<false>(p.m, i0, p.N, mn);                    // sparse steps keep m_t as b- only
    return;
  } else {
    const bool deferred = CLIPT && p.clip;                  // theta on the mask is left to clip_update_kernel
    if (COMPACT && cnt == 0) {
      // no selected entry in this chunk (88 % of the chunks at 99.9 % sparsity): l.6-8 and l.17 only
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const float pq = __fmul_rn(p.b1, mo[q]);
#pragma unroll
        for (int r = 0; r < R; ++r) ee[r][q] = __fadd_rn(__fmaf_rn(p.c1, gg[r][q], pq), ee[r][q]);   // l.6-7
        key0[q] = __float_as_uint(ee[0][q]) & 0x7FFFFFFFu;
        th[q] = __fmaf_rn(p.neg_lr, __fmaf_rn(p.wd, th[q], 0.0f), th[q]);                            // l.17, u = 0 (Eq. 5)
      }
    } else if (!COMPACT || cnt < p.compact_min) {
      // one or two selected entries: l.10-16 in place, on the few lanes that own them
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
        float u = 0.0f;                                                          // Eq. 5: u = 0 off the mask
        if (on) {                                                                // divergent: only the owning lanes run it
          {
            const uint32_t j = jbase + __popc(mybits & ((1u << q) - 1u));
            float* pk = p.packed + j;
            float sm = mt[0];
#pragma unroll
            for (int r = 0; r < R; ++r) { *pk = mt[r]; pk += p.packed_stride; }                 // l.9
#pragma unroll
            for (int r = 1; r < R; ++r) sm = __fadd_rn(sm, mt[r]);                              // l.10, r ascending
            const float bb = p.r_pow2 ? __fmul_rn(sm, p.inv_R) : __fdiv_rn(sm, p.R_f);          // l.10
            const float gh = __fdiv_rn(__fsub_rn(bb, pq), p.c1);                                // l.13 (Eq. 3)
            const float vmq = __fmul_rn(p.b2, __fmul_rn(mo[q], mo[q]));
            p.packed_mean[j] = bb;                                                              // l.12: m_t = b-
            if (deferred) {
              if (p.clip == 2) { p.ghat[j] = sm; p.vm[j] = mo[q]; }
              else {
                p.ghat[j] = gh; p.vm[j] = vmq;
                sa.sumsq += (double)gh * (double)gh;
              }
            } else {
              const float v = __fmaf_rn(p.c2, __fmul_rn(gh, gh), vmq);                          // l.15
              u = __fdiv_rn(__fmul_rn(bb, p.bc1), __fadd_rn(__fsqrt_rn(__fmul_rn(v, p.bc2)), p.eps));   // l.16 (+ :77)
            }
          }
        }
        if (deferred && on) continue;
        th[q] = __fmaf_rn(p.neg_lr, __fmaf_rn(p.wd, th[q], u), th[q]);                         // l.17
      }
    } else {
      const uint32_t lbase = jbase - r0;                    // rank of this lane's first entry inside the chunk
      uint32_t lj = lbase;                                  // walks this lane's selected entries
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
          float* pk = p.packed + (r0 + lj);
          float sm = mt[0];
#pragma unroll
          for (int r = 0; r < R; ++r) { *pk = mt[r]; pk += p.packed_stride; }                   // l.9
#pragma unroll
          for (int r = 1; r < R; ++r) sm = __fadd_rn(sm, mt[r]);                                // l.10, r ascending
          scs[lj] = sm; scm[lj] = mo[q];
          ++lj;
        }
      }
      __syncwarp();
      for (uint32_t l = lane; l < cnt; l += 32) {           // lane l: the chunk's selected entry of rank l
        const float sm = scs[l], mq = scm[l];
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
          scs[l] = __fdiv_rn(__fmul_rn(bb, p.bc1), __fadd_rn(__fsqrt_rn(__fmul_rn(v, p.bc2)), p.eps));   // l.16 (+ :77)
        }
      }
      __syncwarp();
      lj = lbase;
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const bool on = (mybits >> q) & 1u;
        const float u = on ? scs[lj] : 0.0f;                                                   // Eq. 5 off the mask
        lj += on ? 1u : 0u;
        if (deferred && on) continue;
        th[q] = __fmaf_rn(p.neg_lr, __fmaf_rn(p.wd, th[q], u), th[q]);                         // l.17
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
    // Append this chunk's candidates to the warp's segment (their order inside the segment is
    // irrelevant: the composite keys carry the index).  Two forms, chosen by measurement: the
    // register-staged front-end is issue-bound and takes the shorter one (one prefix over the lanes
    // from three ballots on the bits of the per-lane count); the bulk-copy front-end is register-
    // bound (96 registers per thread) and keeps the one with the shortest live ranges.
    if constexpr (STORE) {
      if (__any_sync(0xFFFFFFFFu, cnib != 0u)) {
        const uint32_t n = __popc(cnib), lt = (1u << lane) - 1u;
        const uint32_t b0 = __ballot_sync(0xFFFFFFFFu, n & 1u), b1 = __ballot_sync(0xFFFFFFFFu, n & 2u),
                       b2 = __ballot_sync(0xFFFFFFFFu, n & 4u);
        uint32_t pos = sa.cursor + __popc(b0 & lt) + 2u * __popc(b1 & lt) + 4u * __popc(b2 & lt);
        if (cnib != 0u) {
          const uint32_t inv = 0xFFFFFFFFu - (uint32_t)i0;
          if (pos + 4u <= p.seg_cap) {                      // room for all four: one pointer, no bound checks
            uint2* dst = reinterpret_cast<uint2*>(sa.seg + pos);
#pragma unroll
            for (int q = 0; q < 4; ++q)
              if ((cnib >> q) & 1u) { *dst = make_uint2(inv - q, key0[q]); ++dst; }      // little endian: low word = index part
          } else {
#pragma unroll
            for (int q = 0; q < 4; ++q) {
              if ((cnib >> q) & 1u) {
                if (pos < p.seg_cap) sa.seg[pos] = ((unsigned long long)key0[q] << 32) | (unsigned long long)(inv - q);
                ++pos;
              }
            }
          }
        }
        sa.cursor += __popc(b0) + 2u * __popc(b1) + 4u * __popc(b2);
      }
    } else {
      if (__any_sync(0xFFFFFFFFu, cnib != 0u)) {              // candidates are rare: usually skipped
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
    uint32_t w = nib << ((lane & 7) << 2);
    w |= __shfl_xor_sync(0xFFFFFFFFu, w, 1);
    w |= __shfl_xor_sync(0xFFFFFFFFu, w, 2);
    w |= __shfl_xor_sync(0xFFFFFFFFu, w, 4);
    if ((lane & 7) == 0) p.next_bits[(c << 2) + (lane >> 3)] = w;
  }
}

template <typename G, int R, bool DENSE, bool MSPARSE, bool GUARD, bool CLIPT>
__device__ __forceinline__ void fused_chunk(const StepParams& p, int64_t c, int lane, float* sc, StageA& sa) {
  const int64_t i0 = (c << 7) + ((int64_t)lane << 2);
  // Issue order matters for latency: the mask words first (L2-resident, short latency), then the
  // 2R+1 streaming loads, and only then the gather of m_{t-1}, whose addresses depend on the
  // mask words -- it is in flight together with the streaming loads instead of after them.
  uint4 cw = make_uint4(~0u, ~0u, ~0u, ~0u), pw = make_uint4(0, 0, 0, 0);
  uint32_t cr = 0, pr = 0;
  if (!DENSE) { cw = __ldg(reinterpret_cast<const uint4*>(p.cur_bits) + c); cr = __ldg(p.cur_rank + c); }
  if (MSPARSE) { pw = __ldg(reinterpret_cast<const uint4*>(p.prev_bits) + c); pr = __ldg(p.prev_rank + c); }

  float th[4], mo[4], gg[R][4], ee[R][4];
  load4_f32<GUARD>(p.theta, i0, p.N, th);
  if (!MSPARSE) load4_f32<false>(p.m, i0, p.N, mo);         // own arrays are padded to Npad
#pragma unroll
  for (int r = 0; r < R; ++r) {
    load4_grad<G, GUARD>(p.g[r], i0, p.N, gg[r]);
    load4_f32<false>(p.e + r * p.e_stride, i0, p.N, ee[r]);
  }

  uint32_t mybits = 0xFu, jbase = 0;
  if (!DENSE) lane_bits_from_words(cw, cr, lane, mybits, jbase);
  if (MSPARSE) {
    uint32_t pbits, pbase;
    lane_bits_from_words(pw, pr, lane, pbits, pbase);
    gather_prev_m(p.pm_prev, pbits, pbase, mo);
  }

  fused_compute<R, DENSE, GUARD, true, CLIPT>(p, c, lane, i0, mybits, jbase, cr, DENSE ? 0u : chunk_popc(cw), sc, sc + kChunk, th, mo, gg, ee, sa);
}

template <typename G, int R, bool DENSE, bool MSPARSE, bool CLIPT>
// resident CTAs per SM: sparse steps with one or two replicas are latency-bound (12-24 bytes per parameter in
// flight per lane), so they trade registers for a fourth CTA (measured, N = 2^28, R = 2, 90 %: 2.54 -> 2.29 ms)
__global__ void __launch_bounds__(256, ((!DENSE && R <= 2) ? 4 : R <= 4 ? 3 : 2)) scape_fused_step_kernel(const __grid_constant__ StepParams p) {
  const int lane = threadIdx.x & 31;
  const int64_t wpb = blockDim.x >> 5;
  const int64_t warp = (int64_t)blockIdx.x * wpb + (threadIdx.x >> 5);
  const int64_t nwarps = (int64_t)gridDim.x * wpb;
  const int64_t full = p.N >> 7;
  __shared__ float scratch[DENSE ? 1 : 8 * 2 * kChunk];     // per warp: (sum_r m~^r, m_old) of the selected entries
  float* sc = DENSE ? scratch : scratch + (threadIdx.x >> 5) * (2 * kChunk);
  StageA sa{};
  sa.layer = kNoLayer;
  if (!DENSE) {
    sa.lo = p.ctl->br.lo_key; sa.hi = p.ctl->br.hi_key;
    sa.seg = p.cand + (size_t)warp * p.seg_cap;
  }
  for (int64_t c = warp; c < full; c += nwarps) fused_chunk<G, R, DENSE, MSPARSE, false, CLIPT>(p, c, lane, sc, sa);
  if (full < p.n_chunks && warp == full % nwarps) fused_chunk<G, R, DENSE, MSPARSE, true, CLIPT>(p, full, lane, sc, sa);
  if (!DENSE) {
    if (p.chunk_layer != nullptr) warp_flush_layer(p, sa, lane);      // per-layer counts; seg_above stays 0
    uint32_t na = sa.n_above;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) na += __shfl_xor_sync(0xFFFFFFFFu, na, o);
    if (lane == 0) { p.seg_count[warp] = sa.cursor; p.seg_above[warp] = na; }
  }
  if (CLIPT && p.clip == 1) warp_store_sumsq(p, sa, warp, lane);
}

// ------------------------------------------------------------------------------------------
// Steady-state variant with shared-memory staging (sparse mask in, m stored sparsely).
//
// The LDG kernel above keeps every byte in flight in registers (2R+1 128-bit loads per lane), so
// registers bound the memory-level parallelism (80 regs -> 24 warps/SM -> ~86 KB in flight per
// SM).  Here one producer lane per CTA streams whole tiles of 1024 parameters (theta, e^r, g^r
// slices: 1+2R bulk copies, `cp.async.bulk` = SASS UBLKCP, completion counted in bytes on an
// mbarrier) into a ring of shared-memory stages; 8 consumer warps wait on the stage's "full"
// barrier, pull their 128-bit slices out of shared memory, release the stage ("empty" barrier,
// one arrival per warp) and do the arithmetic and the (fire-and-forget) global stores from
// registers.  Bytes in flight = (stages-1) x tile per CTA, independent of register pressure.
// ------------------------------------------------------------------------------------------
constexpr int kTmaConsumerWarps = 8;
constexpr int kTmaTile = kTmaConsumerWarps * kChunk;          // 1024 parameters
constexpr int kTmaThreads = (kTmaConsumerWarps + 1) * 32;     // + 1 producer warp
constexpr int kTmaMaxStages = 8;
constexpr int kTmaBarrierBytes = 128;                         // full[8] + empty[8]

template <typename G, int R>
__host__ __device__ constexpr uint32_t tma_tile_bytes() { return kTmaTile * 4u * (1u + R) + kTmaTile * (uint32_t)sizeof(G) * R; }

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

struct TmaMaskWords { uint4 cw, pw; uint32_t cr, pr; };
struct TmaTileState { uint32_t mybits, jbase, r0, cnt; float mo[4]; };

__device__ __forceinline__ void tma_load_words(const StepParams& p, int64_t c, TmaMaskWords& w) {
  w.cw = __ldg(reinterpret_cast<const uint4*>(p.cur_bits) + c); w.cr = __ldg(p.cur_rank + c);
  w.pw = __ldg(reinterpret_cast<const uint4*>(p.prev_bits) + c); w.pr = __ldg(p.prev_rank + c);
}
// decode a chunk's mask words for this lane and start the gather of m_{t-1}
__device__ __forceinline__ void tma_decode_gather(const StepParams& p, const TmaMaskWords& w, int lane, TmaTileState& st) {
  uint32_t pbits, pbase;
  lane_bits_from_words(w.cw, w.cr, lane, st.mybits, st.jbase);
  st.r0 = w.cr; st.cnt = chunk_popc(w.cw);
  lane_bits_from_words(w.pw, w.pr, lane, pbits, pbase);
  gather_prev_m(p.pm_prev, pbits, pbase, st.mo);
}

// One tile of one consumer warp: start the next tile's gather, wait for this tile's bytes, pull
// them out of shared memory, release the stage, compute and store.
__device__ __forceinline__ void bulk_s2g(void* dst, const void* src_smem, uint32_t bytes, uint64_t policy) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group.L2::cache_hint [%0], [%1], %2, %3;"
               ::"l"(dst), "r"(smem_u32(src_smem)), "r"(bytes), "l"(policy) : "memory");
}

template <typename G, int R, bool CLIPT>
__device__ __forceinline__ void tma_consume_tile(const StepParams& p, int64_t tile, int64_t n_tiles, int64_t tstride,
                                                 int warp, int lane, unsigned char* stage0, uint64_t* full, uint64_t* empty,
                                                 int& s, uint32_t& ph, int n_stages, TmaMaskWords& nw,
                                                 TmaTileState& cur, TmaTileState& nxt, StageA& sa) {
  constexpr uint32_t TILE = tma_tile_bytes<G, R>();
  constexpr uint32_t OFF_E = kTmaTile * 4u, OFF_G = kTmaTile * 4u * (1u + R);
  const int64_t c = tile * kTmaConsumerWarps + warp;
  const int64_t i0 = (c << 7) + ((int64_t)lane << 2);
  if (tile + tstride < n_tiles) {
    tma_decode_gather(p, nw, lane, nxt);
    if (tile + 2 * tstride < n_tiles) tma_load_words(p, (tile + 2 * tstride) * kTmaConsumerWarps + warp, nw);
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
  // scratch of the on-mask arithmetic: this warp's own theta and e^0 slices of the stage (their
  // contents are in registers now and are written back only after fused_compute)
  unsigned char* wbase = stage0 + (size_t)s * TILE;
  __syncwarp();
  fused_compute<R, false, false, false, CLIPT>(p, c, lane, i0, cur.mybits, cur.jbase, cur.r0, cur.cnt,
                                               reinterpret_cast<float*>(wbase) + warp * kChunk,
                                               reinterpret_cast<float*>(wbase + OFF_E) + warp * kChunk, th, cur.mo, gg, ee, sa);
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
    if (tile != (int64_t)blockIdx.x) mbar_arrive(&empty[s == 0 ? n_stages - 1 : s - 1]);
  }
  if (++s == n_stages) { s = 0; ph ^= 1u; }
}

template <typename G, int R, bool CLIPT>
__global__ void __launch_bounds__(kTmaThreads, 2) scape_fused_tma_kernel(const __grid_constant__ StepParams p, int n_stages) {
  extern __shared__ __align__(128) unsigned char smem[];
  constexpr uint32_t TILE = tma_tile_bytes<G, R>();
  constexpr uint32_t OFF_E = kTmaTile * 4u, OFF_G = kTmaTile * 4u * (1u + R);
  uint64_t* full = reinterpret_cast<uint64_t*>(smem);
  uint64_t* empty = full + kTmaMaxStages;
  unsigned char* stage0 = smem + kTmaBarrierBytes;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int64_t n_tiles = p.N / kTmaTile;                     // full tiles; the rest goes through the LDG path

  if (threadIdx.x == 0) {
    for (int s = 0; s < n_stages; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], 1); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  if (warp == kTmaConsumerWarps) {
    // ===== producer: one lane streams the tiles of this CTA =====
    if (lane == 0) {
      uint64_t policy;
      asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(policy));
      int s = 0; uint32_t ph = 0;
      for (int64_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
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
  const int64_t gwarp = (int64_t)blockIdx.x * kTmaConsumerWarps + warp;     // candidate segment of this warp
  StageA sa{};
  sa.layer = kNoLayer;
  sa.lo = p.ctl->br.lo_key; sa.hi = p.ctl->br.hi_key;
  sa.seg = p.cand + (size_t)gwarp * p.seg_cap;

  // Software pipeline of the small dependent accesses, so that none of their latency is exposed
  // once a tile has landed: mask words are fetched two tiles ahead, and the gather of m_{t-1}
  // (whose addresses come from the previous mask's words) one tile ahead.  The per-tile state
  // ping-pongs between two register sets (A, B) so that no register move has to wait for a load.
  const int64_t tstride = gridDim.x;
  int64_t tile = blockIdx.x;
  TmaMaskWords nw{};                                   // raw words of the NEXT tile
  TmaTileState stA{}, stB{};
  if (tile < n_tiles) {
    TmaMaskWords w0;
    tma_load_words(p, tile * kTmaConsumerWarps + warp, w0);
    if (tile + tstride < n_tiles) tma_load_words(p, (tile + tstride) * kTmaConsumerWarps + warp, nw);
    tma_decode_gather(p, w0, lane, stA);
  }
  int s = 0; uint32_t ph = 0;
  while (tile < n_tiles) {
    tma_consume_tile<G, R, CLIPT>(p, tile, n_tiles, tstride, warp, lane, stage0, full, empty, s, ph, n_stages, nw, stA, stB, sa);
    tile += tstride;
    if (tile >= n_tiles) break;
    tma_consume_tile<G, R, CLIPT>(p, tile, n_tiles, tstride, warp, lane, stage0, full, empty, s, ph, n_stages, nw, stB, stA, sa);
    tile += tstride;
  }
  if (threadIdx.x == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");   // stores have landed
  asm volatile("bar.sync 1, %0;" ::"n"(kTmaConsumerWarps * 32) : "memory");          // ... and every consumer warp knows

  // chunks past the last full tile (fewer than 8, the last one possibly ragged): LDG path
  {
    const int64_t c = n_tiles * kTmaConsumerWarps + warp;
    if (c < p.n_chunks && blockIdx.x == (unsigned)(n_tiles % gridDim.x)) {
      // (all bulk stores of this CTA have completed: the first stage serves as scratch)
      float* sc = reinterpret_cast<float*>(stage0) + warp * (2 * kChunk);
      if (((c + 1) << 7) <= p.N) fused_chunk<G, R, false, true, false, CLIPT>(p, c, lane, sc, sa);
      else fused_chunk<G, R, false, true, true, CLIPT>(p, c, lane, sc, sa);
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
// Stage 2: exact top-k by radix select on the composite 64-bit key
//     K64(i) = bits(|m~^0[i]|) << 32 | (0xFFFFFFFF - i)
// Larger K64 = larger magnitude, ties to the LOWER index (reading S7); all keys are distinct,
// so "the k largest" is unique and selected(i) <=> K64(i) >= T64, T64 the k-th largest.
// The statistic is not stored on its own: off the current mask |m~^0| is exactly the new e^0,
// on it it is b^0 (conservation, pin P2), so the passes re-read those.
// ------------------------------------------------------------------------------------------
struct KeySrc {
  const float* e0;            // [Npad]
  const uint32_t* cur_bits;   // mask the step used (nullptr => treat every position as "off":
  const uint32_t* cur_rank;   //   all-ones step with m~^0 stashed in e^0)
  const float* packed0;       // b^0
  int64_t N;
  int64_t n_chunks;
};

__device__ __forceinline__ unsigned long long make_k64(float x, int64_t i) {
  return ((unsigned long long)(__float_as_uint(x) & 0x7FFFFFFFu) << 32) | (unsigned long long)(0xFFFFFFFFu - (uint32_t)i);
}

// keys of this lane's 4 elements of chunk c (valid[q] false past N)
__device__ __forceinline__ void chunk_keys(const KeySrc& s, int64_t c, int lane, unsigned long long (&k64)[4], bool (&valid)[4]) {
  const int64_t i0 = (c << 7) + ((int64_t)lane << 2);
  const float4 ev = __ldcs(reinterpret_cast<const float4*>(s.e0 + i0));
  float x[4] = {ev.x, ev.y, ev.z, ev.w};
  if (s.cur_bits != nullptr) {
    uint32_t mybits, jbase;
    lane_mask_bits(s.cur_bits, s.cur_rank, c, lane, mybits, jbase);
#pragma unroll
    for (int q = 0; q < 4; ++q)
      if ((mybits >> q) & 1u) x[q] = __ldg(s.packed0 + jbase + __popc(mybits & ((1u << q) - 1u)));
  }
#pragma unroll
  for (int q = 0; q < 4; ++q) { valid[q] = i0 + q < s.N; k64[q] = make_k64(x[q], i0 + q); }
}

// Candidate list written by the fused pass: n_seg segments of seg_cap entries.
constexpr uint32_t kClsCap = 1u << 20;   // entries of the small list the surviving class is collected into

// Scan of the candidate segments by the whole grid.  The fused pass leaves one segment per warp
// (a few thousand of them).  Long segments (large shards: ~10^4 entries each): a work item is one
// of P equal slices of one segment, items are dealt round-robin to the CTAs, and the threads of a
// CTA stride through a slice with 4 independent 8-byte loads each (one warp per segment left two
// thirds of the grid idle and the rest walking long chains of dependent trips).  Short segments
// (small shards: the pass is latency-bound): one warp per segment, all segments at once.
template <typename F>
__device__ __forceinline__ void scan_segments(const unsigned long long* cand, const uint32_t* seg_count, uint32_t seg_cap,
                                              int n_seg, unsigned long long n_cand, F f) {
  if (n_cand <= 256ull * (unsigned long long)n_seg) {
    const int lane = threadIdx.x & 31;
    const int64_t wpb = blockDim.x >> 5;
    const int64_t nwarps = (int64_t)gridDim.x * wpb;
    for (int64_t sg = (int64_t)blockIdx.x * wpb + (threadIdx.x >> 5); sg < n_seg; sg += nwarps) {
      const uint32_t cnt = min(seg_count[sg], seg_cap);
      const unsigned long long* seg = cand + (size_t)sg * seg_cap;
      for (uint32_t j0 = 0; j0 < cnt; j0 += 128) {
        unsigned long long v[4]; bool ok[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) { const uint32_t j = j0 + u * 32 + lane; ok[u] = j < cnt; v[u] = ok[u] ? __ldcs(seg + j) : 0ull; }
#pragma unroll
        for (int u = 0; u < 4; ++u) if (ok[u]) f(v[u]);
      }
    }
    return;
  }
  const uint32_t P = max(1u, (2u * gridDim.x + (uint32_t)n_seg - 1u) / (uint32_t)n_seg);
  const uint32_t n_items = (uint32_t)n_seg * P;
  for (uint32_t it = blockIdx.x; it < n_items; it += gridDim.x) {
    const uint32_t sg = it % (uint32_t)n_seg, part = it / (uint32_t)n_seg;
    const uint32_t cnt = min(seg_count[sg], seg_cap);
    const uint32_t per = ((cnt + P - 1u) / P + 31u) & ~31u;      // slice length, whole 256-byte lines
    const uint32_t b = part * per, e = min(cnt, b + per);
    const unsigned long long* seg = cand + (size_t)sg * seg_cap;
    for (uint32_t j0 = b + threadIdx.x; j0 < e; j0 += 4u * blockDim.x) {
      unsigned long long v[4]; bool ok[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) { const uint32_t j = j0 + u * blockDim.x; ok[u] = j < e; v[u] = ok[u] ? __ldcs(seg + j) : 0ull; }
#pragma unroll
      for (int u = 0; u < 4; ++u) if (ok[u]) f(v[u]);
    }
  }
}

struct CandList {
  unsigned long long* cls;      // [kClsCap] small list (see sel_hist_kernel)
  const unsigned long long* cand;
  const uint32_t* seg_count;
  const uint32_t* seg_above;
  uint32_t seg_cap;
  int n_seg;
};

// One block.  Sums the per-warp counts of the fused pass and decides whether the predicted bracket
// held: hit <=> no segment overflowed and n_above < k <= n_above + n_cand.  Arms the radix select
// with the rank sought inside the candidate list (hit) or inside the whole partition (general).
__global__ void __launch_bounds__(1024) sel_decide_kernel(SelState* st, uint32_t* ghist, CandList cl, long long k, int force_general) {
  __shared__ unsigned long long s_above[32], s_cand[32];
  __shared__ int s_over;
  for (int b = threadIdx.x; b < kBins; b += blockDim.x) ghist[b] = 0;
  if (threadIdx.x == 0) s_over = 0;
  __syncthreads();
  unsigned long long a = 0, c = 0;
  int over = 0;
  if (!force_general) {
    for (int i = threadIdx.x; i < cl.n_seg; i += blockDim.x) {
      const uint32_t cnt = cl.seg_count[i];
      a += cl.seg_above[i]; c += cnt;
      over |= cnt > cl.seg_cap;
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) { a += __shfl_xor_sync(0xFFFFFFFFu, a, o); c += __shfl_xor_sync(0xFFFFFFFFu, c, o); }
  if ((threadIdx.x & 31) == 0) { s_above[threadIdx.x >> 5] = a; s_cand[threadIdx.x >> 5] = c; }
  if (over) s_over = 1;
  __syncthreads();
  if (threadIdx.x == 0) {
    a = 0; c = 0;
    for (int i = 0; i < 32; ++i) { a += s_above[i]; c += s_cand[i]; }
    const bool hit = !force_general && !s_over && (long long)a < k && (long long)(a + c) >= k;
    // On the fast route every candidate key lies in [lo_key, hi_key): the passes run on
    // K64 - (lo_key << 32), whose bits above 32 + ceil(log2(hi_key - lo_key)) are all zero, and start
    // there.  Fewer passes, and the first digit spreads the candidates over at least half of the
    // histogram wherever the bracket sits (skipping only the bits lo and hi share leaves a few
    // hundred crowded bins when the bracket straddles a power of two: contended shared-memory
    // atomics, and a surviving class of 10^5 keys for the second pass to collect).
    unsigned long long prefix0 = 0, himask0 = 0, base = 0;
    int top = 64;
    if (hit) {
      const uint32_t lo = st->br.lo_key, span1 = st->br.hi_key - 1u - lo;      // largest key - lo
      base = (unsigned long long)lo << 32;
      top = 32 + (span1 ? 32 - __clz(span1) : 0);
    }
    st->base = base;
    st->prefix = prefix0; st->himask = himask0; st->top = top;
    st->use_cls = 0; st->cls_n = 0; st->class_count = ~0ull;
    st->rank = hit ? k - (long long)a : k;
    st->hit = hit ? 1 : 0;
    st->n_above = a; st->n_cand = c;
    st->cand_cap_total = (unsigned long long)cl.n_seg * cl.seg_cap;
    if (hit) st->n_fast += 1; else st->n_general += 1;
    if (!hit && !force_general) {
      // too many candidates for the list: narrower next time (a threshold outside the bracket
      // widens it by itself through the prediction error, see sel_pick_kernel)
      if (s_over) st->br.delta = fmaxf(st->br.delta * 0.5f, 0.03f);
    }
  }
}

// Histogram of digit (K64 >> shift) & (2^bits - 1) over the keys whose higher digits equal prefix.
// Source: the small list once the surviving class has been collected into it; else the candidate
// list when the bracket held (st->hit); else every key of the partition.  The pass that first
// sees a class of at most kClsCap keys also collects that class into the small list, so the
// remaining passes touch a few thousand keys instead of re-reading everything.
__global__ void __launch_bounds__(256) sel_hist_kernel(const __grid_constant__ KeySrc s, const __grid_constant__ CandList cl,
                                                      SelState* __restrict__ st, uint32_t* __restrict__ ghist) {
  __shared__ uint32_t h[kBins];
  const int hit = st->hit;
  const int top = st->top;
  if (top <= 0) return;                                   // every digit is fixed already
  const int bits = top < kDigitBits ? top : kDigitBits;
  const int shift = top - bits;
  const int use_cls = st->use_cls;
  const bool collect = !use_cls && st->class_count <= (unsigned long long)kClsCap;
  const uint32_t cls_blocks = min(8u, gridDim.x);         // a handful of CTAs is plenty for the small list
  if (use_cls && blockIdx.x >= cls_blocks) return;
  for (int b = threadIdx.x; b < kBins; b += blockDim.x) h[b] = 0;
  __syncthreads();
  const unsigned long long prefix = st->prefix, himask = st->himask;
  const uint32_t dmask = (1u << bits) - 1u;
  const int lane = threadIdx.x & 31;
  const int64_t wpb = blockDim.x >> 5;
  const int64_t warp = (int64_t)blockIdx.x * wpb + (threadIdx.x >> 5);
  const int64_t nwarps = (int64_t)gridDim.x * wpb;
  const unsigned long long base = st->base;
  auto visit = [&](unsigned long long k64) {
    const unsigned long long kr = k64 - base;
    if ((kr & himask) == prefix) {
      atomicAdd(&h[(uint32_t)(kr >> shift) & dmask], 1u);
      if (collect) { const uint32_t pos = atomicAdd(&st->cls_n, 1u); if (pos < kClsCap) cl.cls[pos] = k64; }
    }
  };
  if (use_cls) {
    const uint32_t n = min(st->cls_n, kClsCap);
    for (uint32_t j = blockIdx.x * blockDim.x + threadIdx.x; j < n; j += cls_blocks * blockDim.x) visit(cl.cls[j]);
  } else if (hit) {
    scan_segments(cl.cand, cl.seg_count, cl.seg_cap, cl.n_seg, st->n_cand, visit);
  } else {
    for (int64_t c = warp; c < s.n_chunks; c += nwarps) {
      unsigned long long k64[4]; bool valid[4];
      chunk_keys(s, c, lane, k64, valid);
#pragma unroll
      for (int q = 0; q < 4; ++q) if (valid[q]) visit(k64[q]);
    }
  }
  __syncthreads();
  for (int b = threadIdx.x; b < kBins; b += blockDim.x) if (h[b]) atomicAdd(&ghist[b], h[b]);
}

// Predict the next step's bracket around the exact threshold just found (the top-k
// structure of the first moment is temporally stable).  The threshold moves smoothly from step to
// step (transient of the EMA, then stationary), so the centre is extrapolated geometrically and the
// half-width follows the error the previous extrapolation made.  shrink > 0: cap the half-width at
// shrink x the old one (the candidate list was more than half full).
__device__ float g_narrow = 0.7f;        // factor by which the half-width may shrink per step (SCAPE_NARROW: experiments; 0.55 missed once in the sweep)
__device__ float g_err_mult = 3.0f;      // half-width >= g_err_mult x the last prediction error + 0.01 (SCAPE_ERR_MULT)
__device__ __forceinline__ void predict_bracket(Bracket& b, uint32_t Tkey, float shrink) {
  const float T = __uint_as_float(Tkey);
  float dl = b.delta, pred;
  if (!(T > 0.0f) || !(T < 3.0e38f)) {           // zero / non-finite threshold: no prediction
    b.lo_key = b.hi_key = 0xFFFFFFFFu; b.have_T = 0;
    return;
  }
  const float lnT = __logf(T);
  if (b.have_T == 0) { pred = lnT; dl = 0.6f; }
  else {
    // Step-to-step change r of ln T.  In the transient of the EMA r decays geometrically,
    // so the next change is predicted as r * (r / r_prev) (ratio clamped to [0, 1]; no
    // extrapolation at all when the sign flips, e.g. for alternating inputs).
    const float r = fminf(fmaxf(lnT - b.lnT_prev, -0.7f), 0.7f);
    float rn = r;
    if (b.have_T >= 2) {
      const float rp = b.r_prev;
      const float ratio = (rp != 0.0f && (r > 0.0f) == (rp > 0.0f)) ? fminf(fmaxf(r / rp, 0.0f), 1.0f) : 0.0f;
      rn = r * ratio;
    }
    pred = lnT + rn;
    b.r_prev = r;
    if (b.have_T == 1) dl = fmaxf(0.05f, 0.5f * fabsf(r));
    else dl = fmaxf(g_err_mult * fabsf(lnT - b.ln_pred) + 0.01f, g_narrow * dl);   // widen at once, narrow slowly
  }
  if (shrink > 0.0f) dl = fminf(dl, b.delta * shrink);
  dl = fminf(fmaxf(dl, 0.02f), 1.0f);
  const float lo = __expf(pred - dl), hi = __expf(pred + dl);
  b.lo_key = __float_as_uint(lo) & 0x7FFFFFFFu;
  b.hi_key = (hi < 3.0e38f) ? (__float_as_uint(hi) & 0x7FFFFFFFu) : 0x7F800000u;
  if (b.hi_key <= b.lo_key) b.hi_key = b.lo_key + 1u;
  b.delta = dl; b.lnT_prev = lnT; b.ln_pred = pred;
  b.have_T = b.have_T < 2 ? b.have_T + 1 : 2;
}

// One block: find the digit d whose class holds the sought rank; fix it; clear the histogram.
__global__ void __launch_bounds__(1024) sel_pick_kernel(SelState* st, uint32_t* ghist) {
  constexpr int PER = kBins / 1024;                 // bins per thread
  const int top_in = st->top;
  if (top_in <= 0) return;
  const int bits = top_in < kDigitBits ? top_in : kDigitBits;
  const int shift = top_in - bits;
  const int last = shift == 0;
  __shared__ long long warp_tot[32];
  const int t = threadIdx.x, lane = t & 31, wid = t >> 5;
  // thread t owns bins [kBins - PER*(t+1), kBins - PER*t): thread 0 owns the TOP bins
  const int top = kBins - PER * t;
  uint32_t hv[PER];
  long long local = 0;
#pragma unroll
  for (int q = 0; q < PER; ++q) { hv[q] = ghist[top - 1 - q]; local += hv[q]; }
  // inclusive prefix sum over threads (from the top bins downwards)
  long long incl = local;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { long long v = __shfl_up_sync(0xFFFFFFFFu, incl, o); if (lane >= o) incl += v; }
  if (lane == 31) warp_tot[wid] = incl;
  __syncthreads();
  if (wid == 0) {
    long long v = warp_tot[lane], iv = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { long long x = __shfl_up_sync(0xFFFFFFFFu, iv, o); if (lane >= o) iv += x; }
    warp_tot[lane] = iv - v;                        // exclusive
  }
  __syncthreads();
  const long long above = warp_tot[wid] + incl - local;   // keys in bins above this thread's bins
  const long long rank = st->rank;
  __syncthreads();
  if (above < rank && rank <= above + local) {
    long long cum = above;
#pragma unroll
    for (int q = 0; q < PER; ++q) {
      if (cum < rank && rank <= cum + hv[q]) {
        const unsigned long long d = (unsigned long long)(top - 1 - q);
        const unsigned long long T64 = st->prefix | (d << shift);
        st->prefix = T64;
        st->himask |= ((1ull << bits) - 1ull) << shift;
        st->rank = rank - cum;
        st->top = shift;
        // the pass that just ran collected its class iff that class was known to be small enough
        if (!st->use_cls && st->class_count <= (unsigned long long)kClsCap) st->use_cls = 1;
        st->class_count = hv[q];
        if (last) {
          // T64 is now exact (back in the key domain): predict the next step's bracket around it
          const unsigned long long Tk = T64 + st->base;
          st->prefix = Tk; st->base = 0;
          float shrink = 0.0f;              // keep the expected candidate count under half the list's capacity
          if (st->hit && st->cand_cap_total > 0 && 2ull * st->n_cand > st->cand_cap_total)
            shrink = (float)st->cand_cap_total / (2.0f * (float)st->n_cand);
          predict_bracket(st->br, (uint32_t)(Tk >> 32), shrink);
        }
      }
      cum += hv[q];
    }
  }
#pragma unroll
  for (int q = 0; q < PER; ++q) ghist[top - 1 - q] = 0;
}

// Complete M_t once T64 (= st->prefix) is exact: selected(i) <=> K64(i) >= T64.
//   bracket held : the fused pass already wrote the certainly-selected bits; OR in the candidates
//   general path : rewrite every word from the keys
__global__ void __launch_bounds__(256) sel_finish_kernel(const __grid_constant__ KeySrc s, const __grid_constant__ CandList cl,
                                                        const SelState* __restrict__ st, uint32_t* __restrict__ next_bits) {
  const unsigned long long T64 = st->prefix;
  const int lane = threadIdx.x & 31;
  const int64_t wpb = blockDim.x >> 5;
  const int64_t warp = (int64_t)blockIdx.x * wpb + (threadIdx.x >> 5);
  const int64_t nwarps = (int64_t)gridDim.x * wpb;
  if (st->hit) {
    scan_segments(cl.cand, cl.seg_count, cl.seg_cap, cl.n_seg, st->n_cand, [&](unsigned long long k64) {
      if (k64 >= T64) {
        const uint32_t i = 0xFFFFFFFFu - (uint32_t)k64;
        atomicOr(&next_bits[i >> 5], 1u << (i & 31));
      }
    });
    return;
  }
  for (int64_t c = warp; c < s.n_chunks; c += nwarps) {
    unsigned long long k64[4]; bool valid[4];
    chunk_keys(s, c, lane, k64, valid);
    uint32_t nib = 0;
#pragma unroll
    for (int q = 0; q < 4; ++q) nib |= (valid[q] && k64[q] >= T64) ? (1u << q) : 0u;
    uint32_t w = nib << ((lane & 7) << 2);
    w |= __shfl_xor_sync(0xFFFFFFFFu, w, 1);
    w |= __shfl_xor_sync(0xFFFFFFFFu, w, 2);
    w |= __shfl_xor_sync(0xFFFFFFFFu, w, 4);
    if ((lane & 7) == 0) next_bits[(c << 2) + (lane >> 3)] = w;
  }
}

// ------------------------------------------------------------------------------------------
// Per-layer refresh ("the top-k sparsification is performed in a per-layer style",
// :138 "number of layers in model L"; uncompressed LayerNorm / RMSNorm / bias layers: :246, :279,
// :286).  The same exact radix select on the same composite keys, run for every layer at once:
// one LayerState per layer, one histogram per layer in global memory.  A layer whose predicted
// bracket held works on the candidates the fused pass collected; the others (no prediction yet,
// a miss, an all-ones step) read their keys back from e^0 / b^0 in work items that never cross a
// layer boundary, so that a CTA can keep a private shared-memory histogram per item.
// ------------------------------------------------------------------------------------------
struct LayerWork {
  const uint32_t* chunk_layer;  // [Npad/128]
  LayerState* layers;
  int n_layers;
  LayerCtl* ctl;
  uint32_t* hist;               // [n_layers][kBins]
  const int4* items;            // {layer, first chunk, end chunk, 0}: <= kItemChunks chunks of one layer
  int n_items;
};
constexpr int kItemChunks = 2048;
constexpr int SCAPE_MAX_LAYERS_K = 4096;           // == SCAPE_MAX_LAYERS (include/scape.h; static_assert in scape.cu)

// Layer of element i by binary search over the layer ends held in shared memory (the candidate
// lists are visited in an order that makes the chunk_layer table, N/32 bytes, a stream of L2
// misses: one random 4-byte load per candidate; the ends are at most 32 KB and stay on chip).
__device__ __forceinline__ void load_layer_ends(const LayerWork& w, long long* ends) {
  for (int l = threadIdx.x; l < w.n_layers; l += blockDim.x) ends[l] = w.layers[l].end;
  __syncthreads();
}
__device__ __forceinline__ uint32_t layer_of_sorted(const long long* ends, int n_layers, uint32_t i) {
  int lo = 0, hi = n_layers - 1;                   // first l with ends[l] > i
  while (lo < hi) {
    const int mid = (lo + hi) >> 1;
    if (ends[mid] > (long long)i) hi = mid; else lo = mid + 1;
  }
  return (uint32_t)lo;
}

__device__ __forceinline__ uint32_t layer_of(const LayerWork& w, uint32_t i) {
  const uint32_t cl = __ldg(w.chunk_layer + (i >> 7));
  uint32_t l = cl & 0x7FFFFFFFu;
  if (cl >> 31) while ((long long)i >= w.layers[l].end) ++l;          // chunk shared by several layers
  return l;
}

// One block.  Per layer: k_l of this refresh (reading S6 inside the layer, evaluated in double
// like the host does), route, and the armed radix state.
__global__ void __launch_bounds__(1024) lsel_decide_kernel(LayerWork w, CandList cl, double sparsity, int force_general) {
  __shared__ unsigned long long s_cand[32];
  __shared__ int s_over;
  if (threadIdx.x == 0) s_over = 0;
  __syncthreads();
  unsigned long long c = 0;
  int over = 0;
  if (!force_general)
    for (int i = threadIdx.x; i < cl.n_seg; i += blockDim.x) { const uint32_t cnt = cl.seg_count[i]; c += cnt; over |= cnt > cl.seg_cap; }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(0xFFFFFFFFu, c, o);
  if ((threadIdx.x & 31) == 0) s_cand[threadIdx.x >> 5] = c;
  if (over) s_over = 1;
  __syncthreads();
  if (threadIdx.x == 0) {
    c = 0;
    for (int i = 0; i < 32; ++i) c += s_cand[i];
    const unsigned long long cap = (unsigned long long)cl.n_seg * cl.seg_cap;
    w.ctl->overflow = s_over;
    w.ctl->shrink = (!force_general && cap > 0 && 2ull * c > cap) ? (float)cap / (2.0f * (float)c) : 0.0f;
    w.ctl->any_general = 0;
    w.ctl->cls_total = 0; w.ctl->cls_n = 0; w.ctl->use_cls = 0;
  }
  __syncthreads();
  unsigned long long nf = 0, ng = 0;
  for (int l = threadIdx.x; l < w.n_layers; l += blockDim.x) {
    LayerState& S = w.layers[l];
    const long long n = S.end - S.begin;
    const long long k = S.compress ? n - (long long)floor(sparsity * (double)n) : n;
    const long long a = (long long)S.n_above;
    S.n_above = 0;
    S.k = k;
    if (S.skip) {            // not this worker's layer: nothing to find, no bit to set (its bracket stays "none")
      S.hit = 1; S.rank = 0; S.top = 0; S.prefix = ~0ull; S.himask = ~0ull; S.base = 0;
      continue;
    }
    const bool predicted = !(S.br.lo_key == 0xFFFFFFFFu && S.br.hi_key == 0xFFFFFFFFu);
    const bool hit = !force_general && !s_over && predicted && a <= k;
    S.hit = hit ? 1 : 0;
    if (hit) {
      nf += 1;
      S.rank = k - a;                                  // still to be found among the layer's candidates
      S.base = 0;
      if (S.rank == 0) { S.top = 0; S.prefix = ~0ull; S.himask = ~0ull; }     // nothing more to select
      else {
        // every candidate of the layer lies in [lo_key, hi_key): the passes run on K64 - (lo_key << 32)
        // and start at the top of that difference (see sel_decide_kernel)
        const uint32_t lo = S.br.lo_key, span1 = S.br.hi_key - 1u - lo;
        S.base = (unsigned long long)lo << 32;
        S.himask = 0; S.prefix = 0;
        S.top = 32 + (span1 ? 32 - __clz(span1) : 0);
      }
    } else {
      ng += 1;
      S.rank = k; S.top = 64; S.prefix = 0; S.himask = 0; S.base = 0;
      atomicOr(&w.ctl->any_general, 1);
      if (!force_general && s_over && S.compress) S.br.delta = fmaxf(S.br.delta * 0.5f, 0.03f);
    }
  }
  if (nf) atomicAdd(&w.ctl->n_fast, nf);
  if (ng) atomicAdd(&w.ctl->n_general, ng);
}

__device__ __forceinline__ bool layer_digit(const LayerState& S, unsigned long long k64, uint32_t& d) {
  const int top = S.top;
  const unsigned long long kr = k64 - S.base;
  if (top <= 0 || (kr & S.himask) != S.prefix) return false;
  const int bits = top < kDigitBits ? top : kDigitBits;
  d = (uint32_t)(kr >> (top - bits)) & ((1u << bits) - 1u);
  return true;
}

// Digit histograms of the layers on the candidate route.  The candidates of one layer fall into a
// handful of bins in the first pass, so equal (layer, digit) pairs of a warp are merged before the
// global atomic.
__global__ void __launch_bounds__(256) lsel_hist_cand_kernel(const __grid_constant__ LayerWork w, const __grid_constant__ CandList cl) {
  __shared__ long long ends[SCAPE_MAX_LAYERS_K];
  load_layer_ends(w, ends);
  const int lane = threadIdx.x & 31;
  const int64_t wpb = blockDim.x >> 5;
  const int64_t warp = (int64_t)blockIdx.x * wpb + (threadIdx.x >> 5);
  const int64_t nwarps = (int64_t)gridDim.x * wpb;
  // small list (LayerCtl): nobody changes these two fields while this kernel runs, so every CTA
  // takes the same decision; lsel_hist_full_kernel's bookkeeping repeats it afterwards
  const bool use_cls = w.ctl->use_cls != 0;
  const unsigned long long ctot = w.ctl->cls_total;
  const bool collect = !use_cls && ctot > 0 && ctot <= (unsigned long long)kClsCap;
  // one warp-wide step: 32 keys (ok = this lane has one), equal (layer, digit) pairs merged
  auto visit32 = [&](bool ok, unsigned long long k64) {
    uint32_t tag = 0xFFFFFFFFu;
    if (ok) {
      const uint32_t l = layer_of_sorted(ends, w.n_layers, 0xFFFFFFFFu - (uint32_t)k64);
      uint32_t d;
      if (w.layers[l].hit && layer_digit(w.layers[l], k64, d)) {
        tag = (l << kDigitBits) | d;
        if (collect) { const uint32_t pos = atomicAdd(&w.ctl->cls_n, 1u); if (pos < kClsCap) cl.cls[pos] = k64; }
      }
    }
    const uint32_t same = __match_any_sync(0xFFFFFFFFu, tag);
    if (tag != 0xFFFFFFFFu && (__ffs(same) - 1) == lane) atomicAdd(&w.hist[tag], (uint32_t)__popc(same));
  };
  if (use_cls) {
    const uint32_t n = min(w.ctl->cls_n, kClsCap);
    for (int64_t j0 = warp * 32; j0 < (int64_t)n; j0 += nwarps * 32) {
      const int64_t j = j0 + lane;
      visit32(j < (int64_t)n, j < (int64_t)n ? cl.cls[j] : 0ull);
    }
    return;
  }
  // work item = one of P equal slices of one segment (see scan_segments), one warp per item
  const uint32_t n_seg = (uint32_t)cl.n_seg;
  const uint32_t P = max(1u, (uint32_t)((4 * nwarps + n_seg - 1) / n_seg));
  for (int64_t it = warp; it < (int64_t)n_seg * P; it += nwarps) {
    const uint32_t sg = (uint32_t)(it % n_seg), part = (uint32_t)(it / n_seg);
    const uint32_t cnt = min(cl.seg_count[sg], cl.seg_cap);
    const uint32_t per = ((cnt + P - 1u) / P + 31u) & ~31u;
    const uint32_t b = part * per, e = min(cnt, b + per);
    const unsigned long long* seg = cl.cand + (size_t)sg * cl.seg_cap;
    for (uint32_t j0 = b; j0 < e; j0 += 32) {
      const uint32_t j = j0 + lane;
      visit32(j < e, j < e ? __ldcs(seg + j) : 0ull);
    }
  }
}

// Digit histograms of the layers on the general route: every key of the layer, item by item.
__global__ void __launch_bounds__(256) lsel_hist_full_kernel(const __grid_constant__ KeySrc s, const __grid_constant__ LayerWork w) {
  __shared__ uint32_t h[kBins];
  // Bookkeeping of the small list, between the candidate pass that just ran and the picks that
  // follow: a pass that was collecting has completed the list; the class sizes are summed afresh.
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    const unsigned long long ctot = w.ctl->cls_total;
    if (!w.ctl->use_cls && ctot > 0 && ctot <= (unsigned long long)kClsCap) w.ctl->use_cls = 1;   // the pass before this copied them
    w.ctl->cls_total = 0;
  }
  if (!w.ctl->any_general) return;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, wpb = blockDim.x >> 5;
  for (int it = blockIdx.x; it < w.n_items; it += gridDim.x) {
    const int4 item = __ldg(w.items + it);
    const LayerState& S = w.layers[item.x];
    if (S.hit || S.top <= 0) continue;                      // block-uniform
    for (int b = threadIdx.x; b < kBins; b += blockDim.x) h[b] = 0;
    __syncthreads();
    const long long lb = S.begin, le = S.end;
    for (int64_t c = item.y + wid; c < item.z; c += wpb) {
      unsigned long long k64[4]; bool valid[4];
      chunk_keys(s, c, lane, k64, valid);
      const int64_t i0 = (c << 7) + ((int64_t)lane << 2);
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        uint32_t d;
        if (valid[q] && i0 + q >= lb && i0 + q < le && layer_digit(S, k64[q], d)) atomicAdd(&h[d], 1u);
      }
    }
    __syncthreads();
    uint32_t* gh = w.hist + (size_t)item.x * kBins;
    for (int b = threadIdx.x; b < kBins; b += blockDim.x) if (h[b]) atomicAdd(&gh[b], h[b]);
    __syncthreads();
  }
}

// One block per layer: find the digit whose class holds the sought rank; fix it; clear the
// layer's histogram.  A layer on the candidate route whose candidates turn out to be fewer than
// the rank sought (the bracket missed) restarts on the general route.
__global__ void __launch_bounds__(1024) lsel_pick_kernel(LayerWork w) {
  constexpr int PER = kBins / 1024;
  LayerState& S = w.layers[blockIdx.x];
  uint32_t* ghist = w.hist + (size_t)blockIdx.x * kBins;
  const int top_in = S.top;
  if (top_in <= 0) return;
  const int bits = top_in < kDigitBits ? top_in : kDigitBits;
  const int shift = top_in - bits;
  __shared__ long long warp_tot[32];
  __shared__ long long s_total;
  const int t = threadIdx.x, lane = t & 31, wid = t >> 5;
  const int topb = kBins - PER * t;                 // thread 0 owns the TOP bins
  uint32_t hv[PER];
  long long local = 0;
#pragma unroll
  for (int q = 0; q < PER; ++q) { hv[q] = ghist[topb - 1 - q]; local += hv[q]; ghist[topb - 1 - q] = 0; }
  long long incl = local;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { long long v = __shfl_up_sync(0xFFFFFFFFu, incl, o); if (lane >= o) incl += v; }
  if (lane == 31) warp_tot[wid] = incl;
  __syncthreads();
  if (wid == 0) {
    long long v = warp_tot[lane], iv = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { long long x = __shfl_up_sync(0xFFFFFFFFu, iv, o); if (lane >= o) iv += x; }
    warp_tot[lane] = iv - v;
    if (lane == 31) s_total = iv;
  }
  __syncthreads();
  const long long above = warp_tot[wid] + incl - local;
  const long long rank = S.rank;
  const long long total = s_total;
  const int hit = S.hit;
  __syncthreads();
  if (total < rank) {
    // only possible on the candidate route, first pass: fewer candidates than entries still to
    // select, i.e. the true threshold lies below the bracket
    if (t == 0) {
      S.hit = 0; S.rank = S.k; S.top = 64; S.prefix = 0; S.himask = 0; S.base = 0;
      atomicOr(&w.ctl->any_general, 1);
      atomicAdd(&w.ctl->n_general, 1ull);
      atomicAdd(&w.ctl->n_fast, ~0ull);              // - 1
    }
    return;
  }
  if (above < rank && rank <= above + local) {
    long long cum = above;
#pragma unroll
    for (int q = 0; q < PER; ++q) {
      if (cum < rank && rank <= cum + hv[q]) {
        const unsigned long long d = (unsigned long long)(topb - 1 - q);
        unsigned long long T64 = S.prefix | (d << shift);
        if (shift == 0) { T64 += S.base; S.base = 0; }       // exact: back in the key domain
        S.prefix = T64;
        S.himask |= ((1ull << bits) - 1ull) << shift;
        S.rank = rank - cum;
        S.top = shift;
        if (hit && shift > 0) atomicAdd(&w.ctl->cls_total, (unsigned long long)hv[q]);   // size of the surviving class
        if (shift == 0 && S.compress) predict_bracket(S.br, (uint32_t)(T64 >> 32), hit ? w.ctl->shrink : 0.0f);
      }
      cum += hv[q];
    }
  }
}

// M_t of the layers on the general route: rewrite every bit of the layer from its keys.
__global__ void __launch_bounds__(256) lsel_finish_full_kernel(const __grid_constant__ KeySrc s, const __grid_constant__ LayerWork w,
                                                              uint32_t* __restrict__ next_bits) {
  if (!w.ctl->any_general) return;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, wpb = blockDim.x >> 5;
  for (int it = blockIdx.x; it < w.n_items; it += gridDim.x) {
    const int4 item = __ldg(w.items + it);
    const LayerState& S = w.layers[item.x];
    if (S.hit) continue;
    const unsigned long long T64 = S.prefix;
    const long long lb = S.begin, le = S.end;
    for (int64_t c = item.y + wid; c < item.z; c += wpb) {
      unsigned long long k64[4]; bool valid[4];
      chunk_keys(s, c, lane, k64, valid);
      const int64_t i0 = (c << 7) + ((int64_t)lane << 2);
      uint32_t nib = 0, own = 0;                            // own: positions of this word that belong to the layer
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const bool in = i0 + q >= lb && i0 + q < le;
        own |= in ? (1u << q) : 0u;
        nib |= (in && valid[q] && k64[q] >= T64) ? (1u << q) : 0u;
      }
      uint32_t v = nib << ((lane & 7) << 2), m = own << ((lane & 7) << 2);
#pragma unroll
      for (int o = 1; o < 8; o <<= 1) { v |= __shfl_xor_sync(0xFFFFFFFFu, v, o); m |= __shfl_xor_sync(0xFFFFFFFFu, m, o); }
      if ((lane & 7) == 0 && m != 0u) {
        uint32_t* wp = next_bits + (c << 2) + (lane >> 3);
        if (m == 0xFFFFFFFFu) *wp = v;
        else { atomicAnd(wp, ~m); atomicOr(wp, v); }       // word shared with a neighbouring layer
      }
    }
  }
}

// M_t of the layers on the candidate route: the fused pass wrote the certainly-selected bits;
// OR in the candidates at or above the layer's threshold.
__global__ void __launch_bounds__(256) lsel_finish_cand_kernel(const __grid_constant__ LayerWork w, const __grid_constant__ CandList cl,
                                                              uint32_t* __restrict__ next_bits) {
  __shared__ long long ends[SCAPE_MAX_LAYERS_K];
  load_layer_ends(w, ends);
  scan_segments(cl.cand, cl.seg_count, cl.seg_cap, cl.n_seg, ~0ull, [&](unsigned long long k64) {
    const uint32_t i = 0xFFFFFFFFu - (uint32_t)k64;
    const LayerState& S = w.layers[layer_of_sorted(ends, w.n_layers, i)];
    if (S.hit && k64 >= S.prefix) atomicOr(&next_bits[i >> 5], 1u << (i & 31));
  });
}

// ------------------------------------------------------------------------------------------
// Ordered compaction of a bit mask: rank128[c] and the ascending index list (the int32 half of
// the sparse buffer).  Three small kernels over N/8 bytes.
// ------------------------------------------------------------------------------------------
constexpr int kCompactChunksPerBlock = 1024;   // one thread per chunk

__global__ void __launch_bounds__(1024) mask_block_count_kernel(const uint32_t* __restrict__ bits, int64_t n_chunks,
                                                               uint32_t* __restrict__ block_sum) {
  __shared__ uint32_t ws[32];
  const int64_t c = (int64_t)blockIdx.x * kCompactChunksPerBlock + threadIdx.x;
  uint32_t n = 0;
  if (c < n_chunks) {
    const uint4 w = __ldg(reinterpret_cast<const uint4*>(bits) + c);
    n = __popc(w.x) + __popc(w.y) + __popc(w.z) + __popc(w.w);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) n += __shfl_xor_sync(0xFFFFFFFFu, n, o);
  if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = n;
  __syncthreads();
  if (threadIdx.x < 32) {
    uint32_t v = ws[threadIdx.x];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, o);
    if (threadIdx.x == 0) block_sum[blockIdx.x] = v;
  }
}

// exclusive scan of block_sum[0..nb) in place, one block; total -> *total_out
__global__ void __launch_bounds__(1024) mask_scan_blocks_kernel(uint32_t* __restrict__ block_sum, int nb, uint32_t* total_out) {
  __shared__ uint32_t ws[32];
  __shared__ uint32_t carry;
  if (threadIdx.x == 0) carry = 0;
  __syncthreads();
  for (int base = 0; base < nb; base += 1024) {
    const int i = base + threadIdx.x;
    const uint32_t v = i < nb ? block_sum[i] : 0u;
    uint32_t incl = v;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { uint32_t x = __shfl_up_sync(0xFFFFFFFFu, incl, o); if (lane >= o) incl += x; }
    if (lane == 31) ws[wid] = incl;
    __syncthreads();
    if (wid == 0) {
      uint32_t x = ws[lane], ix = x;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { uint32_t y = __shfl_up_sync(0xFFFFFFFFu, ix, o); if (lane >= o) ix += y; }
      ws[lane] = ix - x;
    }
    __syncthreads();
    const uint32_t excl = carry + ws[wid] + incl - v;
    if (i < nb) block_sum[i] = excl;
    __syncthreads();
    if (threadIdx.x == 1023) carry = excl + v;
    __syncthreads();
  }
  if (threadIdx.x == 0 && total_out) *total_out = carry;
}

__global__ void __launch_bounds__(1024) mask_rank_idx_kernel(const uint32_t* __restrict__ bits, int64_t n_chunks,
                                                            const uint32_t* __restrict__ block_off,
                                                            uint32_t* __restrict__ rank128, int32_t* __restrict__ idx, int64_t idx_cap) {
  __shared__ uint32_t ws[32];
  const int64_t c = (int64_t)blockIdx.x * kCompactChunksPerBlock + threadIdx.x;
  uint4 w = make_uint4(0, 0, 0, 0);
  if (c < n_chunks) w = __ldg(reinterpret_cast<const uint4*>(bits) + c);
  const uint32_t n = __popc(w.x) + __popc(w.y) + __popc(w.z) + __popc(w.w);
  uint32_t incl = n;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { uint32_t x = __shfl_up_sync(0xFFFFFFFFu, incl, o); if (lane >= o) incl += x; }
  if (lane == 31) ws[wid] = incl;
  __syncthreads();
  if (wid == 0) {
    uint32_t x = ws[lane], ix = x;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { uint32_t y = __shfl_up_sync(0xFFFFFFFFu, ix, o); if (lane >= o) ix += y; }
    ws[lane] = ix - x;
  }
  __syncthreads();
  if (c >= n_chunks) return;
  uint32_t j = block_off[blockIdx.x] + ws[wid] + incl - n;
  rank128[c] = j;
  if (idx == nullptr) return;
  const uint32_t words[4] = {w.x, w.y, w.z, w.w};
  const int64_t base = c << 7;
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    uint32_t x = words[q];
    while (x) {
      const int b = __ffs(x) - 1;
      x &= x - 1;
      if ((int64_t)j < idx_cap) idx[j] = (int32_t)(base + (q << 5) + b);
      ++j;
    }
  }
}

// Single-pass variant of the three kernels above (chained scan with decoupled look-back): every CTA
// takes a ticket (so that all its predecessors have started), scans its 1024 chunk counts,
// publishes its total, looks back over the predecessors' totals / inclusive prefixes until it has its
// own exclusive prefix, publishes the inclusive one and writes rank128 and the index list.  The
// mask bits are read once instead of twice and two launches go away.
//   state[b] = (tag << 32) | value, tag = 2 * epoch + 1: total of block b, 2 * epoch + 2: inclusive
//   prefix through block b; any other tag: nothing yet (epoch changes every call: no clearing).
//   ctl[0] = total number of set bits (out), ctl[1] = ticket (returns to 0).
__global__ void __launch_bounds__(1024) mask_compact_kernel(const uint32_t* __restrict__ bits, int64_t n_chunks,
                                                           unsigned long long* state, uint32_t* ctl, uint32_t epoch,
                                                           uint32_t* __restrict__ rank128, int32_t* __restrict__ idx, int64_t idx_cap) {
  __shared__ uint32_t ws[32];
  __shared__ uint32_t s_bid, s_prefix;
  if (threadIdx.x == 0) s_bid = atomicAdd(&ctl[1], 1u);
  __syncthreads();
  const uint32_t bid = s_bid;
  const int64_t c = (int64_t)bid * 1024 + threadIdx.x;
  uint4 w = make_uint4(0, 0, 0, 0);
  if (c < n_chunks) w = __ldg(reinterpret_cast<const uint4*>(bits) + c);
  const uint32_t n = __popc(w.x) + __popc(w.y) + __popc(w.z) + __popc(w.w);
  uint32_t incl = n;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { uint32_t x = __shfl_up_sync(0xFFFFFFFFu, incl, o); if (lane >= o) incl += x; }
  if (lane == 31) ws[wid] = incl;
  __syncthreads();
  const unsigned long long tag_total = (unsigned long long)(2u * epoch + 1u) << 32, tag_incl = (unsigned long long)(2u * epoch + 2u) << 32;
  if (wid == 0) {
    uint32_t x = ws[lane], ix = x;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { uint32_t y = __shfl_up_sync(0xFFFFFFFFu, ix, o); if (lane >= o) ix += y; }
    ws[lane] = ix - x;
    const uint32_t total = __shfl_sync(0xFFFFFFFFu, ix, 31);
    // publish the total (block 0: already the inclusive prefix), then look back, 32 predecessors at a time
    volatile unsigned long long* vs = state;
    if (lane == 0) { vs[bid] = (bid == 0 ? tag_incl : tag_total) | total; __threadfence(); }
    uint32_t prefix = 0;
    if (bid > 0) {
      int64_t b0 = (int64_t)bid - 1;                    // newest predecessor not yet accounted for
      while (true) {
        const int64_t b = b0 - lane;
        unsigned long long v = 0;
        bool ready, is_incl;
        do {                                            // wait until every predecessor in the window has published
          v = b >= 0 ? vs[b] : tag_incl;                // before block 0: an inclusive prefix of 0
          const unsigned long long tg = v & 0xFFFFFFFF00000000ull;
          is_incl = tg == tag_incl;
          ready = is_incl || tg == tag_total;
        } while (!__all_sync(0xFFFFFFFFu, ready));
        const uint32_t incl_mask = __ballot_sync(0xFFFFFFFFu, is_incl);
        // lanes 0 .. first inclusive one (nearest predecessors first) contribute
        const int stop = incl_mask ? __ffs(incl_mask) - 1 : 31;
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
      if (bid == gridDim.x - 1) { ctl[0] = prefix + total; ctl[1] = 0; }     // every CTA has its ticket by now
    }
  }
  __syncthreads();
  if (c >= n_chunks) return;
  uint32_t j = s_prefix + ws[wid] + incl - n;
  rank128[c] = j;
  if (idx == nullptr) return;
  const uint32_t words[4] = {w.x, w.y, w.z, w.w};
  const int64_t base = c << 7;
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    uint32_t x = words[q];
    while (x) {
      const int b = __ffs(x) - 1;
      x &= x - 1;
      if ((int64_t)j < idx_cap) idx[j] = (int32_t)(base + (q << 5) + b);
      ++j;
    }
  }
}

// ------------------------------------------------------------------------------------------
// l.14 clip_grad (optional, reading S3'): global-norm clip of the reconstructed gradient
// ------------------------------------------------------------------------------------------
struct ClipState { double norm; float coef; int pad; };

// one block: sum the per-warp partial sums in a fixed order, derive the factor
__global__ void __launch_bounds__(1024) clip_norm_kernel(const double* __restrict__ sumsq, int n_slots, double max_norm, ClipState* out) {
  __shared__ double sh[1024];
  double a = 0.0;
  for (int i = threadIdx.x; i < n_slots; i += 1024) a += sumsq[i];
  sh[threadIdx.x] = a;
  __syncthreads();
  for (int o = 512; o > 0; o >>= 1) { if ((int)threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o]; __syncthreads(); }
  if (threadIdx.x == 0) {
    const double nrm = sqrt(sh[0]);
    const double cc = max_norm / (nrm + 1e-6);              // the torch / Megatron clip_grad_norm rule
    out->norm = nrm;
    out->coef = cc < 1.0 ? (float)cc : 1.0f;
  }
}

// l.14-17 for the K entries of the mask: scale g^, second moment, update, parameter step
__global__ void __launch_bounds__(256) clip_update_kernel(float* __restrict__ theta, const int32_t* __restrict__ idx,
                                                         const float* __restrict__ bb, const float* __restrict__ ghat,
                                                         const float* __restrict__ vm, int64_t K, const ClipState* __restrict__ cs,
                                                         float c2, float eps, float wd, float neg_lr, float bc1, float bc2) {
  const float coef = cs->coef;
  for (int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; j < K; j += (int64_t)gridDim.x * blockDim.x) {
    const int64_t i = idx ? (int64_t)idx[j] : j;
    const float gh = __fmul_rn(ghat[j], coef);                                              // l.14
    const float v = __fmaf_rn(c2, __fmul_rn(gh, gh), vm[j]);                               // l.15
    const float u = __fdiv_rn(__fmul_rn(bb[j], bc1), __fadd_rn(__fsqrt_rn(__fmul_rn(v, bc2)), eps));   // l.16 (+ :77)
    const float t = theta[i];
    theta[i] = __fmaf_rn(neg_lr, __fmaf_rn(wd, t, u), t);                                   // l.17
  }
}

// scatter / gather helpers for the dense <-> packed views used by the accessors
// Workers ("all-reduce", §8(f) rank 3): l.10 and l.12-17 for the K selected entries once
// the workers' sums have been added up.  S[j] = sum over ALL R_total replicas of m~^r at idx[j]
// (each worker's own replicas in order, then the workers: the oracle's two-level sum), mold[j] =
// m_{t-1} there.  Same pinned operation order as fused_compute.  idx == nullptr: all-ones step.
__global__ void __launch_bounds__(256) dist_update_kernel(float* __restrict__ theta, const int32_t* __restrict__ idx,
                                                         float* __restrict__ m_out, const float* __restrict__ S,
                                                         const float* __restrict__ mold, int64_t K, float R_f, float inv_R,
                                                         int r_pow2, float b1, float c1, float b2, float c2, float eps, float wd,
                                                         float neg_lr, float bc1, float bc2) {
  // 4 entries per thread and trip: the gather of theta depends on the index load, so the loads of
  // four entries are issued together (one entry per trip left the kernel latency-bound)
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t j0 = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; j0 < K; j0 += 4 * stride) {
    int64_t i[4]; float sm[4], mo[4], th[4]; bool ok[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int64_t j = j0 + u * stride;
      ok[u] = j < K;
      i[u] = ok[u] ? (idx ? (int64_t)__ldg(idx + j) : j) : 0;
      sm[u] = ok[u] ? __ldcs(S + j) : 0.0f;
      mo[u] = ok[u] ? __ldcs(mold + j) : 0.0f;
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) th[u] = ok[u] ? theta[i[u]] : 0.0f;
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      if (!ok[u]) continue;
      const float pq = __fmul_rn(b1, mo[u]);
      const float bb = r_pow2 ? __fmul_rn(sm[u], inv_R) : __fdiv_rn(sm[u], R_f);               // l.10
      const float gh = __fdiv_rn(__fsub_rn(bb, pq), c1);                                       // l.13 (Eq. 3)
      const float v = __fmaf_rn(c2, __fmul_rn(gh, gh), __fmul_rn(b2, __fmul_rn(mo[u], mo[u])));   // l.15
      const float uu = __fdiv_rn(__fmul_rn(bb, bc1), __fadd_rn(__fsqrt_rn(__fmul_rn(v, bc2)), eps));   // l.16 (+ :77)
      theta[i[u]] = __fmaf_rn(neg_lr, __fmaf_rn(wd, th[u], uu), th[u]);                        // l.17
      m_out[j0 + u * stride] = bb;                                                             // l.12: m_t = b- (packed, or dense when idx == nullptr)
    }
  }
}

__global__ void fill_u32_kernel(uint32_t* p, int64_t n, uint32_t v) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) p[i] = v;
}

__global__ void iota_i32_kernel(int32_t* p, int64_t n) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) p[i] = (int32_t)i;
}

// dense[idx[j]] = packed[j]  (dense view of a sparsely stored m, for the accessors)
__global__ void scatter_packed_kernel(float* __restrict__ dense, const int32_t* __restrict__ idx,
                                      const float* __restrict__ packed, int64_t count) {
  for (int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; j < count; j += (int64_t)gridDim.x * blockDim.x)
    dense[idx[j]] = packed[j];
}

// ------------------------------------------------------------------------------------------
// Mask bit pack / unpack ("we convert the masks from INT8 to 1-bit values and pack
// 8 mask values into one byte"; the paper's Triton kernels).  The bit-packed form -- bit i % 32 of
// word i / 32 -- is this library's native mask; these two kernels convert to and from one byte
// per parameter for callers that keep masks that way.  HBM-bound: N bytes on one side, N/8 on the
// other; a thread handles one word = 32 mask values (two independent 16-byte accesses).
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t nonzero_bytes_to_bits16(const uint4 t) {
  const uint32_t x[4] = {t.x, t.y, t.z, t.w};
  uint32_t v = 0;
#pragma unroll
  for (int q = 0; q < 4; ++q)
#pragma unroll
    for (int b = 0; b < 4; ++b) v |= ((x[q] >> (8 * b)) & 0xFFu) ? (1u << (4 * q + b)) : 0u;
  return v;
}
__device__ __forceinline__ uint4 bits16_to_bytes(uint32_t v) {
  uint32_t x[4];
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    const uint32_t n4 = (v >> (4 * q)) & 0xFu;
    x[q] = (n4 & 1u) | ((n4 & 2u) << 7) | ((n4 & 4u) << 14) | ((n4 & 8u) << 21);
  }
  return make_uint4(x[0], x[1], x[2], x[3]);
}

__global__ void __launch_bounds__(256) mask_pack_kernel(const uint8_t* __restrict__ bytes, int64_t N, uint32_t* __restrict__ words) {
  const int64_t n_words = (N + 31) >> 5;
  const bool aligned = ((uintptr_t)bytes & 15) == 0;
  for (int64_t w = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; w < n_words; w += (int64_t)gridDim.x * blockDim.x) {
    const int64_t i0 = w << 5;
    uint32_t v = 0;
    if (aligned && i0 + 32 <= N) {
      const uint4 lo = __ldcs(reinterpret_cast<const uint4*>(bytes + i0));
      const uint4 hi = __ldcs(reinterpret_cast<const uint4*>(bytes + i0 + 16));
      v = nonzero_bytes_to_bits16(lo) | (nonzero_bytes_to_bits16(hi) << 16);
    } else {
      for (int b = 0; b < 32; ++b) if (i0 + b < N && bytes[i0 + b]) v |= 1u << b;
    }
    words[w] = v;
  }
}

// a thread writes 16 values (one 16-byte store; two stores of 32-byte stride per lane wrote half sectors)
__global__ void __launch_bounds__(256) mask_unpack_kernel(const uint32_t* __restrict__ words, int64_t N, uint8_t* __restrict__ bytes) {
  const int64_t n_half = (N + 15) >> 4;
  const bool aligned = ((uintptr_t)bytes & 15) == 0;
  for (int64_t g = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; g < n_half; g += (int64_t)gridDim.x * blockDim.x) {
    const int64_t i0 = g << 4;
    const uint32_t v = (__ldg(words + (g >> 1)) >> ((g & 1) << 4)) & 0xFFFFu;
    if (aligned && i0 + 16 <= N) __stcs(reinterpret_cast<uint4*>(bytes + i0), bits16_to_bytes(v));
    else for (int b = 0; b < 16; ++b) if (i0 + b < N) bytes[i0 + b] = (uint8_t)((v >> b) & 1u);
  }
}

// all-ones mask over [0,N), zero padding bits up to n_words*32
__global__ void mask_all_ones_kernel(uint32_t* bits, int64_t n_words, int64_t N) {
  for (int64_t w = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; w < n_words; w += (int64_t)gridDim.x * blockDim.x) {
    const int64_t lo = w << 5;
    uint32_t v = 0;
    if (lo + 32 <= N) v = 0xFFFFFFFFu;
    else if (lo < N) v = (1u << (uint32_t)(N - lo)) - 1u;
    bits[w] = v;
  }
}

// clear bits at positions >= N (after a user-supplied mask was copied in)
__global__ void mask_clear_tail_kernel(uint32_t* bits, int64_t n_words, int64_t N) {
  for (int64_t w = (N >> 5) + (int64_t)blockIdx.x * blockDim.x + threadIdx.x; w < n_words; w += (int64_t)gridDim.x * blockDim.x) {
    const int64_t lo = w << 5;
    if (lo >= N) bits[w] = 0;
    else bits[w] &= (1u << (uint32_t)(N - lo)) - 1u;
  }
}

}  // namespace scapek
