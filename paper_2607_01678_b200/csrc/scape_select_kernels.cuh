// scape_select_kernels.cuh — the kernels of the SCAPE step that are not the streaming pass: the exact
// top-k select of stage 2 (Alg. 1 l.11), the ordered compaction of a bit mask into
// the position tables (pre, trank) + the ascending index list (the int32 half of the sparse buffer, l.9), the deferred
// updates (clip_grad l.14, workers l.10-17), the mask bit pack / unpack and the
// Algorithm 2 parameter kernels.  Plain (non-template) kernels: this header is
// included by scape.cu only.
#pragma once
#include "scape_kernels.cuh"

namespace scapek {

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
  const uint2* cur_rk;        //   all-ones step with m~^0 stashed in e^0)
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
    lane_mask_bits(s.cur_bits, s.cur_rk, c, lane, mybits, jbase);
#pragma unroll
    for (int q = 0; q < 4; ++q)
      if ((mybits >> q) & 1u) x[q] = __ldg(s.packed0 + jbase + __popc(mybits & ((1u << q) - 1u)));
  }
#pragma unroll
  for (int q = 0; q < 4; ++q) { valid[q] = i0 + q < s.N; k64[q] = make_k64(x[q], i0 + q); }
}

// Candidate list written by the fused pass: n_seg segments of seg_cap entries.
constexpr uint32_t kClsCap = 1u << 20;   // entries of the small list the surviving class is collected into
constexpr uint32_t kClsDirect = 4096;    // a small list of at most this many entries is histogrammed by one CTA with global atomics
constexpr uint32_t kClsDirectLayers = 1u << 16;   // per-layer select: by ceil(n / 256) CTAs

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
  uint32_t rec_seg_cap;         // layout of the recovery pass's candidate segments (SelState::rec)
  int rec_n_seg;
};

// One block.  Sums the per-warp counts of the fused pass and decides whether the predicted bracket
// held: hit <=> no segment overflowed and n_above < k <= n_above + n_cand.  Arms the radix select
// with the rank sought inside the candidate list (hit) or inside the whole partition (general).
//   fused: the streaming kernel has added the histogram of the candidates' first digit (kFusedBits bits) to
//   ghist whenever fused_hist_shift(bracket) >= 0; it is kept if the bracket held and cleared otherwise.
__global__ void __launch_bounds__(1024) sel_decide_kernel(SelState* st, uint32_t* ghist, CandList cl, long long k, int force_general, int fused) {
  __shared__ unsigned long long s_above[32], s_cand[32];
  __shared__ int s_over, s_keep;
  if (threadIdx.x == 0) { s_over = 0; s_keep = 0; }
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
    const bool keep = hit && fused && fused_hist_shift(st->br.lo_key, st->br.hi_key) >= 0;
    st->first_bits = keep ? (unsigned int)kFusedBits : 0u;
    s_keep = keep ? 1 : 0;
    st->base = base;
    st->prefix = prefix0; st->himask = himask0; st->top = top;
    st->use_cls = 0; st->cls_n = 0; st->class_count = ~0ull; st->bits_done = 0;
    st->rank = hit ? k - (long long)a : k;
    st->hit = hit ? 1 : 0;
    st->need_rec = hit ? 0 : 1;                     // a miss (or no bracket at all): try the recovery pass before the general route
    st->rec = 0;
    st->n_above = a; st->n_cand = c;
    st->cand_cap_total = (unsigned long long)cl.n_seg * cl.seg_cap;
    if (hit) st->n_fast += 1; else st->n_general += 1;
    if (!hit && !force_general) {
      // too many candidates for the list: narrower next time (a threshold outside the bracket
      // widens it by itself through the prediction error, see sel_pick_kernel)
      if (s_over) st->br.delta = fmaxf(st->br.delta * 0.5f, 0.03f);
    }
  }
  __syncthreads();
  if (!s_keep) for (int b = threadIdx.x; b < kBins; b += blockDim.x) ghist[b] = 0;
}

// ------------------------------------------------------------------------------------------
// Recovery of a missed bracket, and the select of an all-ones step (SelState::need_rec).  The general
// route re-reads every key three to five times (8.9 ms on the headline shard, a ~26 ms step).  Instead:
//   sel_sample_kernel       histogram of the top 13 key bits over every 64th chunk (every chunk of small shards)
//   sel_sample_pick_kernel  the bin holding the (scaled) k-th largest sampled key; bracket = that bin
//                           widened by a quarter bin on either side: [lo2, hi2)
//   sel_classify_kernel     ONE pass over every key: key >= hi2 sets its bit of M_t, lo2 <= key < hi2
//                           joins the candidate list (own segment layout), the rest is dropped
//   sel_decide2_kernel      n_above < k <= n_above + n_cand and no overflow?  then the candidate route
//                           takes over (rec = 1); else the general route runs as before
// Exactness does not depend on the sample: it is the same check as for the predicted bracket.
// All four return at once when the predicted bracket held.
// ------------------------------------------------------------------------------------------
constexpr int kRecStride = 64;            // large shards: every 64th chunk is sampled; at least ~2048 chunks (2.6e5 keys) always
__host__ __device__ __forceinline__ int64_t rec_stride(int64_t n_chunks) {
  const int64_t s = n_chunks / 2048;
  return s < 1 ? 1 : s > kRecStride ? kRecStride : s;
}
constexpr int kRecShift = 32 - kDigitBits;  // digit of the sample histogram = key >> 19 (exponent + 4 mantissa bits)

__global__ void __launch_bounds__(256) sel_sample_kernel(const __grid_constant__ KeySrc s, const SelState* __restrict__ st,
                                                        uint32_t* __restrict__ ghist) {
  if (!st->need_rec) return;
  __shared__ uint32_t h[kBins];
  for (int b = threadIdx.x; b < kBins; b += blockDim.x) h[b] = 0;
  __syncthreads();
  const int lane = threadIdx.x & 31;
  const int64_t wpb = blockDim.x >> 5;
  const int64_t warp = (int64_t)blockIdx.x * wpb + (threadIdx.x >> 5);
  const int64_t nwarps = (int64_t)gridDim.x * wpb;
  const int64_t stride = rec_stride(s.n_chunks);
  for (int64_t c = warp * stride; c < s.n_chunks; c += nwarps * stride) {
    unsigned long long k64[4]; bool valid[4];
    chunk_keys(s, c, lane, k64, valid);
#pragma unroll
    for (int q = 0; q < 4; ++q) if (valid[q]) atomicAdd(&h[(uint32_t)(k64[q] >> (32 + kRecShift))], 1u);
  }
  __syncthreads();
  for (int b = threadIdx.x; b < kBins; b += blockDim.x) if (h[b]) atomicAdd(&ghist[b], h[b]);
}

// one block of 1024 threads; clears ghist again
__global__ void __launch_bounds__(1024) sel_sample_pick_kernel(SelState* st, uint32_t* ghist, long long k, long long N) {
  if (!st->need_rec) return;
  constexpr int PER = kBins / 1024;
  __shared__ long long warp_tot[32];
  __shared__ long long s_total;
  const int t = threadIdx.x, lane = t & 31, wid = t >> 5;
  const int top = kBins - PER * t;                  // thread 0 owns the TOP bins
  uint32_t hv[PER];
  long long local = 0;
#pragma unroll
  for (int q = 0; q < PER; ++q) { hv[q] = ghist[top - 1 - q]; local += hv[q]; ghist[top - 1 - q] = 0; }
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
  const long long total = s_total;                  // sampled keys
  if (t == 0) { st->lo2 = 0xFFFFFFFFu; st->hi2 = 0xFFFFFFFFu; }
  __syncthreads();
  if (total <= 0) return;
  // rank of the k-th largest key among the sampled ones, by proportion (the sample is every 64th chunk)
  long long ks = (long long)((double)k * (double)total / (double)N);
  if (ks < 1) ks = 1;
  if (ks > total) ks = total;
  if (above < ks && ks <= above + local) {
    long long cum = above;
#pragma unroll
    for (int q = 0; q < PER; ++q) {
      if (cum < ks && ks <= cum + hv[q]) {
        const uint32_t d = (uint32_t)(top - 1 - q);
        const uint32_t edge = d << kRecShift, quarter = 1u << (kRecShift - 2);
        st->lo2 = edge > quarter ? edge - quarter : 0u;
        const unsigned long long hi = (unsigned long long)edge + (1ull << kRecShift) + quarter;
        st->hi2 = hi < 0x7F800000ull ? (uint32_t)hi : 0x7F800000u;
      }
      cum += hv[q];
    }
  }
}

// launched with exactly cl.rec_n_seg warps: warp w owns segment w
__global__ void __launch_bounds__(256, 5) sel_classify_kernel(const __grid_constant__ KeySrc s, const __grid_constant__ CandList cl,
                                                          const SelState* __restrict__ st, unsigned long long* __restrict__ cand,
                                                          uint32_t* __restrict__ seg_count, uint32_t* __restrict__ seg_above,
                                                          uint32_t* __restrict__ next_bits) {
  if (!st->need_rec) return;
  const uint32_t lo = st->lo2, hi = st->hi2;
  if (lo == 0xFFFFFFFFu && hi == 0xFFFFFFFFu) return;      // no bracket from the sample
  const int lane = threadIdx.x & 31;
  const int64_t wpb = blockDim.x >> 5;
  const int64_t warp = (int64_t)blockIdx.x * wpb + (threadIdx.x >> 5);
  const int64_t nwarps = (int64_t)gridDim.x * wpb;
  unsigned long long* seg = cand + (size_t)warp * cl.rec_seg_cap;
  uint32_t cursor = 0, na = 0;
  const LaneMap lm = lane_map(lane);
  // (a lean form of chunk_keys: 32-bit keys only, the mask of the step decoded only in chunks that have
  // selected entries, composite keys built for candidates only: 163 -> ~70 warp instructions per chunk)
  for (int64_t c = warp; c < s.n_chunks; c += nwarps) {
    const uint32_t i0 = (uint32_t)(c << 7) + ((uint32_t)lane << 2);
    const float4 ev = __ldcs(reinterpret_cast<const float4*>(s.e0 + i0));
    float x[4] = {ev.x, ev.y, ev.z, ev.w};
    if (s.cur_bits != nullptr) {
      const uint2 rk = __ldg(s.cur_rk + c);
      if ((rk.y >> 24) != 0u) {                             // warp-uniform: this chunk has entries on the step's mask: their keys are b^0
        uint32_t mybits, jbase;
        lane_decode(__ldg(s.cur_bits + (c << 2) + lm.ws), rk, lm, mybits, jbase);
        const float* pk = s.packed0 + jbase;
#pragma unroll
        for (int q = 0; q < 4; ++q) if ((mybits >> q) & 1u) { x[q] = __ldg(pk); ++pk; }
      }
    }
    const bool last = c == s.n_chunks - 1;
    uint32_t nib = 0, cnib = 0, key[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      key[q] = __float_as_uint(x[q]) & 0x7FFFFFFFu;
      const bool valid = !last || (int64_t)i0 + q < s.N;
      const bool above = valid && key[q] >= hi;
      nib |= above ? (1u << q) : 0u;
      cnib |= (valid && !above && key[q] >= lo) ? (1u << q) : 0u;
    }
    if (__any_sync(0xFFFFFFFFu, cnib != 0u)) {                // candidates are a few per cent of the keys
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const bool cnd = (cnib >> q) & 1u;
        const uint32_t bal = __ballot_sync(0xFFFFFFFFu, cnd);
        if (cnd) {
          const uint32_t pos = cursor + __popc(bal & ((1u << lane) - 1u));
          if (pos < cl.rec_seg_cap) seg[pos] = ((unsigned long long)key[q] << 32) | (unsigned long long)(0xFFFFFFFFu - (i0 + q));
        }
        cursor += __popc(bal);
      }
    }
    na += __popc(nib);
    uint32_t w = nib << lm.sh;
    w |= __shfl_xor_sync(0xFFFFFFFFu, w, 1);
    w |= __shfl_xor_sync(0xFFFFFFFFu, w, 2);
    w |= __shfl_xor_sync(0xFFFFFFFFu, w, 4);
    if (lm.sh == 0u) next_bits[(c << 2) + lm.ws] = w;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) na += __shfl_xor_sync(0xFFFFFFFFu, na, o);
  if (lane == 0) { seg_count[warp] = cursor; seg_above[warp] = na; }
}

// one block: did the sampled bracket hold?
__global__ void __launch_bounds__(1024) sel_decide2_kernel(SelState* st, CandList cl, long long k) {
  if (!st->need_rec) return;
  __shared__ unsigned long long s_above[32], s_cand[32];
  __shared__ int s_over;
  if (threadIdx.x == 0) s_over = 0;
  __syncthreads();
  const uint32_t lo = st->lo2, hi = st->hi2;
  const bool have = !(lo == 0xFFFFFFFFu && hi == 0xFFFFFFFFu);
  unsigned long long a = 0, c = 0;
  int over = 0;
  if (have)
    for (int i = threadIdx.x; i < cl.rec_n_seg; i += blockDim.x) {
      const uint32_t cnt = cl.seg_count[i];
      a += cl.seg_above[i]; c += cnt;
      over |= cnt > cl.rec_seg_cap;
    }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) { a += __shfl_xor_sync(0xFFFFFFFFu, a, o); c += __shfl_xor_sync(0xFFFFFFFFu, c, o); }
  if ((threadIdx.x & 31) == 0) { s_above[threadIdx.x >> 5] = a; s_cand[threadIdx.x >> 5] = c; }
  if (over) s_over = 1;
  __syncthreads();
  if (threadIdx.x == 0) {
    a = 0; c = 0;
    for (int i = 0; i < 32; ++i) { a += s_above[i]; c += s_cand[i]; }
    const bool hit = have && !s_over && (long long)a < k && (long long)(a + c) >= k;
    st->need_rec = 0;
    if (hit) {
      const uint32_t span1 = hi - 1u - lo;
      st->base = (unsigned long long)lo << 32;
      st->top = 32 + (span1 ? 32 - __clz(span1) : 0);
      st->prefix = 0; st->himask = 0;
      st->use_cls = 0; st->cls_n = 0; st->class_count = ~0ull; st->bits_done = 0;
      st->rank = k - (long long)a;
      st->hit = 1; st->rec = 1;
      st->n_above = a; st->n_cand = c;
      st->n_recovered += 1;
    }
    // else: the state sel_decide_kernel armed for the general route stands
  }
}

// Histogram of digit (K64 >> shift) & (2^bits - 1) over the keys whose higher digits equal prefix.
// Source: the small list once the surviving class has been collected into it; else the candidate
// list when the bracket held (st->hit); else every key of the partition.  The pass that first
// sees a class of at most kClsCap keys also collects that class into the small list, so the
// remaining passes touch a few thousand keys instead of re-reading everything.
// On the candidate route that collecting pass also completes M_t for everything outside the class: a
// candidate whose fixed digits lie ABOVE the threshold's is selected whatever the remaining digits
// turn out to be, so its bit is set here and sel_finish_kernel is left with the small list (one pass
// over the whole candidate list less: SelState::bits_done).
__global__ void __launch_bounds__(256) sel_hist_kernel(const __grid_constant__ KeySrc s, const __grid_constant__ CandList cl,
                                                      SelState* __restrict__ st, uint32_t* __restrict__ ghist,
                                                      uint32_t* __restrict__ next_bits) {
  __shared__ uint32_t h[kBins];
  const int hit = st->hit;
  const int top = st->top;
  if (top <= 0) return;                                   // every digit is fixed already
  if (st->first_bits != 0u) return;                       // this digit's histogram came with the streaming kernel
  const int bits = top < kDigitBits ? top : kDigitBits;
  const int shift = top - bits;
  const int use_cls = st->use_cls;
  const bool collect = !use_cls && st->class_count <= (unsigned long long)kClsCap;
  const uint32_t cls_blocks = min(8u, gridDim.x);         // a handful of CTAs is plenty for the small list
  if (use_cls && blockIdx.x >= cls_blocks) return;
  const unsigned long long prefix = st->prefix, himask = st->himask;
  const uint32_t dmask = (1u << bits) - 1u;
  if (use_cls && st->cls_n <= kClsDirect) {
    // a few keys (the usual case from the third digit on: composite keys are distinct, so a class that shares
    // 23 bits holds a handful): one CTA, straight to the global histogram -- clearing and merging a private
    // histogram of 8192 counters was most of such a pass
    if (blockIdx.x != 0) return;
    const unsigned long long base = st->base;
    const uint32_t n = st->cls_n;
    for (uint32_t j = threadIdx.x; j < n; j += blockDim.x) {
      const unsigned long long kr = cl.cls[j] - base;
      if ((kr & himask) == prefix) atomicAdd(&ghist[(uint32_t)(kr >> shift) & dmask], 1u);
    }
    return;
  }
  for (int b = threadIdx.x; b < kBins; b += blockDim.x) h[b] = 0;
  __syncthreads();
  const int lane = threadIdx.x & 31;
  const int64_t wpb = blockDim.x >> 5;
  const int64_t warp = (int64_t)blockIdx.x * wpb + (threadIdx.x >> 5);
  const int64_t nwarps = (int64_t)gridDim.x * wpb;
  const unsigned long long base = st->base;
  const bool set_above = collect && hit;
  auto visit = [&](unsigned long long k64) {
    const unsigned long long kr = k64 - base;
    if ((kr & himask) == prefix) {
      atomicAdd(&h[(uint32_t)(kr >> shift) & dmask], 1u);
      if (collect) { const uint32_t pos = atomicAdd(&st->cls_n, 1u); if (pos < kClsCap) cl.cls[pos] = k64; }
    } else if (set_above && (kr & himask) > prefix) {
      const uint32_t i = 0xFFFFFFFFu - (uint32_t)k64;
      atomicOr(&next_bits[i >> 5], 1u << (i & 31));
    }
  };
  if (use_cls) {
    const uint32_t n = min(st->cls_n, kClsCap);
    for (uint32_t j = blockIdx.x * blockDim.x + threadIdx.x; j < n; j += cls_blocks * blockDim.x) visit(cl.cls[j]);
  } else if (hit) {
    scan_segments(cl.cand, cl.seg_count, st->rec ? cl.rec_seg_cap : cl.seg_cap, st->rec ? cl.rec_n_seg : cl.n_seg, st->n_cand, visit);
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
constexpr float kNarrow = 0.7f;          // factor by which the half-width may shrink per step (measured: 0.55 missed once in the config-5 sweep, 0.85 kept ~1.5x more candidates)
constexpr float kErrMult = 3.0f;         // half-width >= kErrMult x the last prediction error + kErrAdd
constexpr float kErrAdd = 0.004f;        // (0.01 and a floor of 0.02 until round 2: twice the candidates in steady state, where the
constexpr float kMinDelta = 0.008f;      //  prediction error is 0.001-0.003; replayed on the recorded thresholds of 11 workloads: no miss)
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
    else dl = fmaxf(kErrMult * fabsf(lnT - b.ln_pred) + kErrAdd, kNarrow * dl);   // widen at once, narrow slowly
  }
  if (shrink > 0.0f) dl = fminf(dl, b.delta * shrink);
  dl = fminf(fmaxf(dl, kMinDelta), 1.0f);
  const float lo = __expf(pred - dl), hi = __expf(pred + dl);
  b.lo_key = __float_as_uint(lo) & 0x7FFFFFFFu;
  b.hi_key = (hi < 3.0e38f) ? (__float_as_uint(hi) & 0x7FFFFFFFu) : 0x7F800000u;
  if (b.hi_key <= b.lo_key) b.hi_key = b.lo_key + 1u;
  b.delta = dl; b.lnT_prev = lnT; b.ln_pred = pred;
  b.have_T = b.have_T < 2 ? b.have_T + 1 : 2;
}

// Block-wide scan of the kBins counters of ghist from the TOP bin downwards by NT threads: thread t owns the
// PER = kBins / NT bins [kBins - PER (t + 1), kBins - PER t), returned top-down (hv[q] = bin kBins - PER t - 1 - q);
// above = keys in the bins above the thread's, local = keys in its bins, total = all keys.  Clears the histogram.
// Counts fit 32 bits: a pass counts a key of the partition at most once and N < 2^31.
template <int NT>
__device__ __forceinline__ void pick_scan(uint32_t* __restrict__ ghist, uint32_t (&hv)[kBins / NT], uint32_t& above, uint32_t& local,
                                          uint32_t& total) {
  constexpr int PER = kBins / NT;
  static_assert(PER % 4 == 0 && NT % 32 == 0 && NT <= 1024, "pick_scan: whole 16-byte loads per thread");
  __shared__ uint32_t warp_tot[32];
  __shared__ uint32_t s_total;
  const int t = threadIdx.x, lane = t & 31, wid = t >> 5;
  uint4* g4 = reinterpret_cast<uint4*>(ghist + (kBins - PER * (t + 1)));
  uint32_t asc[PER];
#pragma unroll
  for (int j = 0; j < PER / 4; ++j) { const uint4 v = g4[j]; asc[4 * j] = v.x; asc[4 * j + 1] = v.y; asc[4 * j + 2] = v.z; asc[4 * j + 3] = v.w; }
#pragma unroll
  for (int j = 0; j < PER / 4; ++j) g4[j] = make_uint4(0u, 0u, 0u, 0u);
  local = 0;
#pragma unroll
  for (int q = 0; q < PER; ++q) { hv[q] = asc[PER - 1 - q]; local += hv[q]; }
  uint32_t incl = local;                            // inclusive prefix sum over the threads (from the top bins downwards)
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const uint32_t v = __shfl_up_sync(0xFFFFFFFFu, incl, o); if (lane >= o) incl += v; }
  if (lane == 31) warp_tot[wid] = incl;
  __syncthreads();
  if (wid == 0) {
    const uint32_t v = lane < NT / 32 ? warp_tot[lane] : 0u;
    uint32_t iv = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const uint32_t x = __shfl_up_sync(0xFFFFFFFFu, iv, o); if (lane >= o) iv += x; }
    warp_tot[lane] = iv - v;                        // exclusive
    if (lane == 31) s_total = iv;
  }
  __syncthreads();
  above = warp_tot[wid] + incl - local;
  total = s_total;
}

// One block: find the digit d whose class holds the sought rank; fix it; clear the histogram.
// (What the pick needs of the state is loaded together with the histogram: one memory latency instead
// of a chain of six in the thread that finds the digit.)
__global__ void __launch_bounds__(1024) sel_pick_kernel(SelState* st, uint32_t* ghist) {
  constexpr int NT = 1024, PER = kBins / NT;        // bins per thread
  const int top_in = st->top;
  const int fb = (int)st->first_bits;               // a first digit of fb bits, histogrammed by the streaming kernel
  const long long rank = st->rank;
  const unsigned long long prefix = st->prefix, himask = st->himask, base = st->base;
  const unsigned long long class_count = st->class_count, cap_total = st->cand_cap_total, n_cand = st->n_cand;
  const int use_cls = st->use_cls, hit = st->hit, rec = st->rec;
  if (top_in <= 0) return;
  const int bits = fb ? fb : top_in < kDigitBits ? top_in : kDigitBits;
  const int shift = top_in - bits;
  const int last = shift == 0;
  uint32_t hv[PER], above, local, total;
  pick_scan<NT>(ghist, hv, above, local, total);
  const int top = kBins - PER * (int)threadIdx.x;   // this thread's bins end here
  if ((long long)above < rank && rank <= (long long)above + (long long)local) {
    long long cum = above;
#pragma unroll
    for (int q = 0; q < PER; ++q) {
      if (cum < rank && rank <= cum + (long long)hv[q]) {
        const unsigned long long d = (unsigned long long)(top - 1 - q);
        const unsigned long long T64 = prefix | (d << shift);
        st->prefix = T64;
        st->himask = himask | (((1ull << bits) - 1ull) << shift);
        st->rank = rank - cum;
        st->top = shift;
        st->first_bits = 0u;
        // the pass that just ran collected its class iff that class was known to be small enough
        if (!use_cls && class_count <= (unsigned long long)kClsCap) { st->use_cls = 1; st->bits_done = hit; }
        st->class_count = hv[q];
        if (last) {
          // T64 is now exact (back in the key domain): predict the next step's bracket around it
          const unsigned long long Tk = T64 + base;
          st->prefix = Tk; st->base = 0;
          float shrink = 0.0f;              // keep the expected candidate count under half the list's capacity
          if (hit && !rec && cap_total > 0 && 2ull * n_cand > cap_total) shrink = (float)cap_total / (2.0f * (float)n_cand);
          predict_bracket(st->br, (uint32_t)(Tk >> 32), shrink);
        }
      }
      cum += hv[q];
    }
  }
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
  if (st->hit && st->bits_done) {
    // everything above the collected class has its bit already (sel_hist_kernel): the class itself is left
    const uint32_t n = min(st->cls_n, kClsCap);
    for (uint32_t j = blockIdx.x * blockDim.x + threadIdx.x; j < n; j += gridDim.x * blockDim.x) {
      const unsigned long long k64 = cl.cls[j];
      if (k64 >= T64) {
        const uint32_t i = 0xFFFFFFFFu - (uint32_t)k64;
        atomicOr(&next_bits[i >> 5], 1u << (i & 31));
      }
    }
    return;
  }
  if (st->hit) {
    scan_segments(cl.cand, cl.seg_count, st->rec ? cl.rec_seg_cap : cl.seg_cap, st->rec ? cl.rec_n_seg : cl.n_seg, st->n_cand, [&](unsigned long long k64) {
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
// (layer ends fit 32 bits: shard_numel < 2^31.)  `lite`: what a candidate's digit needs of its layer's
// state, for the first kLiteLayers layers, so that a candidate costs shared-memory reads only (the
// LayerState in global memory was five dependent L2 loads per candidate).
constexpr int kLiteLayers = 512;
struct LayerLite { unsigned long long base, himask, prefix; int top; int hit; };
__device__ __forceinline__ LayerLite layer_lite(const LayerState& S) {
  LayerLite L; L.base = S.base; L.himask = S.himask; L.prefix = S.prefix; L.top = S.top; L.hit = S.hit;
  return L;
}
__device__ __forceinline__ void load_layer_ends(const LayerWork& w, uint32_t* ends, LayerLite* lite) {
  for (int l = threadIdx.x; l < w.n_layers; l += blockDim.x) {
    ends[l] = (uint32_t)w.layers[l].end;
    if (l < kLiteLayers) lite[l] = layer_lite(w.layers[l]);
  }
  __syncthreads();
}
// hint: the layer of the previous candidate this thread saw (a segment is in ascending chunk order, so
// the layer rarely changes: one or two comparisons instead of a 12-step search)
__device__ __forceinline__ uint32_t layer_of_sorted(const uint32_t* ends, int n_layers, uint32_t i, uint32_t hint = 0) {
  if (i < ends[hint] && (hint == 0u || i >= ends[hint - 1u])) return hint;
  int lo = 0, hi = n_layers - 1;                   // first l with ends[l] > i
  while (lo < hi) {
    const int mid = (lo + hi) >> 1;
    if (ends[mid] > i) hi = mid; else lo = mid + 1;
  }
  return (uint32_t)lo;
}
// Walking a slice of a segment, 32 consecutive candidates per warp step: the chunks ascend along the slice, so a
// candidate's layer is the one of the candidate before it (hint: the layer of the last lane of the step before, the
// same for all lanes) or one of the next few -- a scan of a step or two instead of a search whose eight dependent
// shared-memory reads were 43 % of the stall samples of the first candidate pass.  (Inside a chunk the order is
// arbitrary, hence the backward loop.)  kNoHint: start of a slice, search.
constexpr uint32_t kNoHint = 0xFFFFFFFFu;
__device__ __forceinline__ uint32_t layer_near(const uint32_t* ends, int n_layers, uint32_t i, uint32_t hint) {
  if (hint == kNoHint) return layer_of_sorted(ends, n_layers, i, 0u);
  uint32_t l = hint;
  while (l > 0u && i < ends[l - 1u]) --l;
  while (l + 1u < (uint32_t)n_layers && i >= ends[l]) ++l;
  return l;
}
__device__ __forceinline__ bool lite_digit(const LayerLite& S, unsigned long long k64, uint32_t& d) {
  const int top = S.top;
  const unsigned long long kr = k64 - S.base;
  if (top <= 0 || (kr & S.himask) != S.prefix) return false;
  const int bits = top < kDigitBits ? top : kDigitBits;
  d = (uint32_t)(kr >> (top - bits)) & ((1u << bits) - 1u);
  return true;
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
    w.ctl->cls_total = 0; w.ctl->cls_n = 0; w.ctl->use_cls = 0; w.ctl->bits_done = 0;
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

// Digit histograms of the layers on the candidate route: one global atomic per candidate of a live
// class (merging equal (layer, digit) pairs of a warp with __match_any_sync first cost more than the
// atomics it saved: first pass 511 -> 437 us on the headline shard without it).
// The pass that collects the small list also sets the bit of every candidate that lies above its layer's
// class (or at / above a threshold that is complete already): see sel_hist_kernel, LayerCtl::bits_done.
__global__ void __launch_bounds__(256) lsel_hist_cand_kernel(const __grid_constant__ LayerWork w, const __grid_constant__ CandList cl,
                                                            uint32_t* __restrict__ next_bits) {
  __shared__ uint32_t ends[SCAPE_MAX_LAYERS_K];
  __shared__ LayerLite lite[kLiteLayers];
  if (w.ctl->use_cls != 0 && w.ctl->cls_n <= kClsDirectLayers) {
    // a few keys per layer (see sel_hist_kernel; a few hundred layers together: 10^3 .. 10^4): one thread per key,
    // the layer from the chunk table, no layer tables in shared memory; the other CTAs return at once (with every
    // CTA loading the tables first, such a pass took 25 us on the headline shard)
    const uint32_t n = w.ctl->cls_n;
    if (blockIdx.x * blockDim.x >= n) return;
    for (uint32_t j = blockIdx.x * blockDim.x + threadIdx.x; j < n; j += gridDim.x * blockDim.x) {
      const unsigned long long k64 = cl.cls[j];
      const uint32_t l = layer_of(w, 0xFFFFFFFFu - (uint32_t)k64);
      const LayerState& S = w.layers[l];
      uint32_t d;
      if (S.hit && layer_digit(S, k64, d)) atomicAdd(&w.hist[(l << kDigitBits) | d], 1u);
    }
    return;
  }
  load_layer_ends(w, ends, lite);
  const int lane = threadIdx.x & 31;
  const int64_t wpb = blockDim.x >> 5;
  const int64_t warp = (int64_t)blockIdx.x * wpb + (threadIdx.x >> 5);
  const int64_t nwarps = (int64_t)gridDim.x * wpb;
  uint32_t hint = 0;
  // small list (LayerCtl): nobody changes these two fields while this kernel runs, so every CTA
  // takes the same decision; lsel_hist_full_kernel's bookkeeping repeats it afterwards
  const bool use_cls = w.ctl->use_cls != 0;
  const unsigned long long ctot = w.ctl->cls_total;
  const bool collect = !use_cls && ctot > 0 && ctot <= (unsigned long long)kClsCap;
  // one warp-wide step: 32 keys (ok = this lane has one)
  // sorted: the keys come from a slice of a segment (hint = warp-uniform, see layer_near); else from the small list,
  // in no order (hint = this lane's previous layer)
  auto visit32 = [&](bool ok, unsigned long long k64, bool sorted) {
    uint32_t tag = 0xFFFFFFFFu;
    uint32_t l = hint;
    if (ok) {
      const uint32_t i = 0xFFFFFFFFu - (uint32_t)k64;
      l = sorted ? layer_near(ends, w.n_layers, i, hint) : layer_of_sorted(ends, w.n_layers, i, hint);
      const LayerLite L = l < (uint32_t)kLiteLayers ? lite[l] : layer_lite(w.layers[l]);
      uint32_t d;
      if (L.hit && lite_digit(L, k64, d)) {
        tag = (l << kDigitBits) | d;
        if (collect) { const uint32_t pos = atomicAdd(&w.ctl->cls_n, 1u); if (pos < kClsCap) cl.cls[pos] = k64; }
      } else if (collect && L.hit) {
        // outside the layer's class: selected iff above it; a layer whose threshold is complete (top == 0:
        // prefix is the threshold itself, base 0; ~0 when the layer has nothing left to select) decides here
        const bool sel = L.top > 0 ? ((k64 - L.base) & L.himask) > L.prefix : k64 >= L.prefix;
        if (sel) { const uint32_t i = 0xFFFFFFFFu - (uint32_t)k64; atomicOr(&next_bits[i >> 5], 1u << (i & 31)); }
      }
    }
    hint = sorted ? __shfl_sync(0xFFFFFFFFu, l, 31) : l;     // a lane without a key keeps the hint it had
    if (tag != 0xFFFFFFFFu) atomicAdd(&w.hist[tag], 1u);
  };
  if (use_cls) {
    const uint32_t n = min(w.ctl->cls_n, kClsCap);
    for (int64_t j0 = warp * 32; j0 < (int64_t)n; j0 += nwarps * 32) {
      const int64_t j = j0 + lane;
      visit32(j < (int64_t)n, j < (int64_t)n ? cl.cls[j] : 0ull, false);
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
    hint = kNoHint;
    for (uint32_t j0 = b; j0 < e; j0 += 128) {            // four independent loads per lane in flight
      unsigned long long v[4]; bool ok[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) { const uint32_t j = j0 + u * 32 + lane; ok[u] = j < e; v[u] = ok[u] ? __ldcs(seg + j) : 0ull; }
#pragma unroll
      for (int u = 0; u < 4; ++u) if (j0 + u * 32 < e) visit32(ok[u], v[u], true);
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
    if (!w.ctl->use_cls && ctot > 0 && ctot <= (unsigned long long)kClsCap) { w.ctl->use_cls = 1; w.ctl->bits_done = 1; }   // the pass before this copied them
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
constexpr int kLayerPickThreads = 512;              // two resident CTAs per SM: a few hundred layers are one wave
__global__ void __launch_bounds__(kLayerPickThreads, 2) lsel_pick_kernel(LayerWork w) {
  constexpr int NT = kLayerPickThreads, PER = kBins / NT;
  LayerState& S = w.layers[blockIdx.x];
  uint32_t* ghist = w.hist + (size_t)blockIdx.x * kBins;
  const int top_in = S.top;
  const long long rank = S.rank;
  const int hit = S.hit;
  const unsigned long long prefix = S.prefix, himask = S.himask, base = S.base;
  if (top_in <= 0) return;
  const int bits = top_in < kDigitBits ? top_in : kDigitBits;
  const int shift = top_in - bits;
  const int t = threadIdx.x;
  const int topb = kBins - PER * t;                 // thread 0 owns the TOP bins
  uint32_t hv[PER], above, local, total;
  pick_scan<NT>(ghist, hv, above, local, total);
  if ((long long)total < rank) {
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
  if ((long long)above < rank && rank <= (long long)above + (long long)local) {
    long long cum = above;
#pragma unroll
    for (int q = 0; q < PER; ++q) {
      if (cum < rank && rank <= cum + (long long)hv[q]) {
        const unsigned long long d = (unsigned long long)(topb - 1 - q);
        unsigned long long T64 = prefix | (d << shift);
        if (shift == 0) { T64 += base; S.base = 0; }         // exact: back in the key domain
        S.prefix = T64;
        S.himask = himask | (((1ull << bits) - 1ull) << shift);
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
  __shared__ uint32_t ends[SCAPE_MAX_LAYERS_K];
  __shared__ LayerLite lite[kLiteLayers];
  if (w.ctl->bits_done) {
    // the collecting pass has set every bit outside the layers' classes: the small list is left
    const uint32_t n = min(w.ctl->cls_n, kClsCap);
    for (uint32_t j = blockIdx.x * blockDim.x + threadIdx.x; j < n; j += gridDim.x * blockDim.x) {
      const unsigned long long k64 = cl.cls[j];
      const uint32_t i = 0xFFFFFFFFu - (uint32_t)k64;
      const LayerState& S = w.layers[layer_of(w, i)];
      if (S.hit && k64 >= S.prefix) atomicOr(&next_bits[i >> 5], 1u << (i & 31));
    }
    return;
  }
  load_layer_ends(w, ends, lite);
  uint32_t hint = 0;
  scan_segments(cl.cand, cl.seg_count, cl.seg_cap, cl.n_seg, ~0ull, [&](unsigned long long k64) {
    const uint32_t i = 0xFFFFFFFFu - (uint32_t)k64;
    const uint32_t l = hint = layer_of_sorted(ends, w.n_layers, i, hint);
    const bool sel = l < (uint32_t)kLiteLayers ? (lite[l].hit && k64 >= lite[l].prefix) : (w.layers[l].hit && k64 >= w.layers[l].prefix);
    if (sel) atomicOr(&next_bits[i >> 5], 1u << (i & 31));
  });
}

// ------------------------------------------------------------------------------------------
// Ordered compaction of a bit mask: rank128[c] and the ascending index list (the int32 half of
// the sparse buffer).  Three small kernels over N/8 bytes.
// ------------------------------------------------------------------------------------------
constexpr int kCompactChunksPerBlock = 1024;   // one thread per chunk

// block_sum[b] = set bits of block b (1024 chunks); warp_pre[c >> 5] = set bits of the block's chunks before the
// group of 32 chunks that c belongs to -- with it mask_rank_idx_kernel needs no block-wide step
// (256 threads, four chunks each, loaded together: one 16-byte load per thread and two CTAs of 1024 per SM kept
// 32 KB per SM in flight, 3.7 TB/s on the headline shard.)
constexpr int kCountThreads = 256;
__global__ void __launch_bounds__(kCountThreads) mask_block_count_kernel(const uint32_t* __restrict__ bits, int64_t n_chunks,
                                                               uint32_t* __restrict__ block_sum, uint32_t* __restrict__ warp_pre) {
  constexpr int U = kCompactChunksPerBlock / kCountThreads;
  __shared__ uint32_t ws[32];
  const int64_t c0 = (int64_t)blockIdx.x * kCompactChunksPerBlock + threadIdx.x;
  uint4 w[U];
#pragma unroll
  for (int u = 0; u < U; ++u) {
    const int64_t c = c0 + u * kCountThreads;
    w[u] = make_uint4(0, 0, 0, 0);
    if (c < n_chunks) w[u] = __ldg(reinterpret_cast<const uint4*>(bits) + c);
  }
#pragma unroll
  for (int u = 0; u < U; ++u) {
    uint32_t n = __popc(w[u].x) + __popc(w[u].y) + __popc(w[u].z) + __popc(w[u].w);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) n += __shfl_xor_sync(0xFFFFFFFFu, n, o);
    if ((threadIdx.x & 31) == 0) ws[(threadIdx.x >> 5) + u * (kCountThreads / 32)] = n;     // group of chunks c >> 5 inside the block
  }
  __syncthreads();
  if (threadIdx.x < 32) {
    const uint32_t v = ws[threadIdx.x];
    uint32_t iv = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const uint32_t x = __shfl_up_sync(0xFFFFFFFFu, iv, o); if ((int)threadIdx.x >= o) iv += x; }
    warp_pre[(size_t)blockIdx.x * 32 + threadIdx.x] = iv - v;
    if (threadIdx.x == 31) block_sum[blockIdx.x] = iv;
  }
}

// exclusive scan of block_sum[0..nb) in place, one block; total -> *total_out.  Thread t owns the
// ceil(nb / 1024) consecutive sums from t * per on and loads them all at once (one memory latency; a loop
// over slabs of 1024 sums was 14 dependent round trips on the headline shard, 15 us).  nb <= 2^14: a
// shard has fewer than 2^24 chunks (N < 2^31) and a block of the count kernel takes 1024 of them.
constexpr int kScanMaxPer = 16;
__global__ void __launch_bounds__(1024) mask_scan_blocks_kernel(uint32_t* __restrict__ block_sum, int nb, uint32_t* total_out) {
  __shared__ uint32_t ws[32];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const int per = (nb + 1023) >> 10;
  const int i0 = (int)threadIdx.x * per;
  uint32_t v[kScanMaxPer], sum = 0;
#pragma unroll
  for (int q = 0; q < kScanMaxPer; ++q) v[q] = (q < per && i0 + q < nb) ? block_sum[i0 + q] : 0u;
#pragma unroll
  for (int q = 0; q < kScanMaxPer; ++q) sum += v[q];
  uint32_t incl = sum;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const uint32_t x = __shfl_up_sync(0xFFFFFFFFu, incl, o); if (lane >= o) incl += x; }
  if (lane == 31) ws[wid] = incl;
  __syncthreads();
  if (wid == 0) {
    const uint32_t x = ws[lane];
    uint32_t ix = x;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const uint32_t y = __shfl_up_sync(0xFFFFFFFFu, ix, o); if (lane >= o) ix += y; }
    ws[lane] = ix - x;
  }
  __syncthreads();
  uint32_t run = ws[wid] + incl - sum;
#pragma unroll
  for (int q = 0; q < kScanMaxPer; ++q) {
    if (q < per && i0 + q < nb) block_sum[i0 + q] = run;
    run += v[q];
  }
  if (threadIdx.x == 1023 && total_out) *total_out = run;
}

// The ascending index list of one chunk per thread (w: the chunk's 128 bits, n of them set, j: packed
// position of the first, c: chunk number).  Sparse chunks: the thread walks its set bits.  Dense chunks
// (more than 32 set bits: a flat top-k concentrates the mask in a few tensors, whose chunks are nearly
// full) would keep one lane looping 128 times while 31 wait, and write 32 runs 500 bytes apart per
// instruction (llama500m at 90 %: 472 us for 50 M indices); the warp takes them one by one instead,
// lane l writing the positions of bits 4l .. 4l+3, so one instruction writes consecutive positions.
// Must be called by whole warps (idx != nullptr is warp-uniform).
__device__ __forceinline__ void write_chunk_indices(const uint4 w, const uint32_t n, uint32_t j, const int64_t c,
                                                    int32_t* __restrict__ idx, const int64_t idx_cap) {
  if (idx == nullptr) return;
  const int lane = threadIdx.x & 31;
  const bool dense = n > 32u;
  if (!dense) {
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
  uint32_t dm = __ballot_sync(0xFFFFFFFFu, dense);
  while (dm) {
    const int src = __ffs(dm) - 1;
    dm &= dm - 1;
    const uint4 ws4 = make_uint4(__shfl_sync(0xFFFFFFFFu, w.x, src), __shfl_sync(0xFFFFFFFFu, w.y, src),
                                 __shfl_sync(0xFFFFFFFFu, w.z, src), __shfl_sync(0xFFFFFFFFu, w.w, src));
    const uint32_t j0 = __shfl_sync(0xFFFFFFFFu, j, src);
    uint32_t mybits, pos;
    lane_bits_from_words(ws4, j0, lane, mybits, pos);
    const int32_t e0 = (int32_t)(((c - lane + src) << 7) + (lane << 2));
#pragma unroll
    for (int q = 0; q < 4; ++q)
      if ((mybits >> q) & 1u) { if ((int64_t)pos < idx_cap) idx[pos] = e0 + q; ++pos; }
  }
}

// One thread per chunk, a warp per group of 32 chunks; the packed position of a group's first set bit is
// block_off[block] + warp_pre[group], so the warps are independent: no shared memory, no barrier (with a
// block-wide scan in here the CTAs alternated between a load phase and a write phase, two per SM:
// 2.6 TB/s on the headline shard).
// The index list leaves through shared memory: the lanes' runs are laid down at their position inside the group's
// run and the warp copies that out 128 bytes per instruction (straight from the lanes every index was a 4-byte
// store to a sector of its own: 27 M L2 write transactions for 107 MB at N = 2^28, 90 %).  Groups with more than
// kStageIdx set bits (dense regions of a flat top-k) write directly; their dense chunks are coalesced already.
// (Several groups per warp, loaded together, were slower: the index writes bound the kernel, not the loads.)
constexpr int kRankIdxThreads = 256;
constexpr int kRankIdxGroups = 2;               // groups of 32 chunks per warp, loaded together
constexpr uint32_t kStageIdx = 1024;
__global__ void __launch_bounds__(kRankIdxThreads) mask_rank_idx_kernel(const uint32_t* __restrict__ bits, int64_t n_chunks,
                                                            const uint32_t* __restrict__ block_off, const uint32_t* __restrict__ warp_pre,
                                                            uint2* __restrict__ rk, uint32_t* __restrict__ pre, uint32_t* __restrict__ trank,
                                                            int32_t* __restrict__ idx, int64_t idx_cap) {
  __shared__ int32_t stage[kRankIdxThreads / 32][kStageIdx];
  const int lane = threadIdx.x & 31;
  const int64_t g0 = ((int64_t)blockIdx.x * (kRankIdxThreads / 32) + (threadIdx.x >> 5)) * kRankIdxGroups;   // this warp's first group
  uint4 w[kRankIdxGroups];
  uint32_t offs[kRankIdxGroups];
#pragma unroll
  for (int u = 0; u < kRankIdxGroups; ++u) {
    const int64_t g = g0 + u, c = (g << 5) + lane;
    w[u] = make_uint4(0, 0, 0, 0);
    offs[u] = 0;
    if (c < n_chunks) w[u] = __ldg(reinterpret_cast<const uint4*>(bits) + c);
    if ((g << 5) < n_chunks) offs[u] = __ldg(block_off + (g >> 5)) + __ldg(warp_pre + g);      // warp-uniform
  }
#pragma unroll
  for (int u = 0; u < kRankIdxGroups; ++u) {
    const int64_t c = ((g0 + u) << 5) + lane;
    if (c - lane >= n_chunks) break;                         // whole warp past the end
    const uint32_t off = offs[u];
    const uint32_t n = __popc(w[u].x) + __popc(w[u].y) + __popc(w[u].z) + __popc(w[u].w);
    uint32_t incl = n;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const uint32_t x = __shfl_up_sync(0xFFFFFFFFu, incl, o); if (lane >= o) incl += x; }
    const uint32_t j = off + incl - n;
    if (c < n_chunks) {
      const uint32_t pb = chunk_prefix_bytes(__popc(w[u].x), __popc(w[u].y), __popc(w[u].z), __popc(w[u].w));
      rk[c] = make_uint2(j, pb);
      pre[c] = pb;
      if ((c & 7) == 0) trank[c >> 3] = j;
      if (c == n_chunks - 1) trank[(c >> 3) + 1] = j + n;    // the table's last entry: every set bit
    }
    if (idx == nullptr) continue;
    const uint32_t total = __shfl_sync(0xFFFFFFFFu, incl, 31); // set bits of the group (past the end: w = 0, n = 0)
    if (total <= kStageIdx) {
      int32_t* sm = stage[threadIdx.x >> 5];
      write_chunk_indices(w[u], n, incl - n, c, sm, (int64_t)kStageIdx);
      __syncwarp();
      for (uint32_t t = lane; t < total; t += 32) {
        const uint32_t pos = off + t;
        if ((int64_t)pos < idx_cap) idx[pos] = sm[t];
      }
      __syncwarp();                                            // the stage is reused by the warp's next group
    } else {
      write_chunk_indices(w[u], n, j, c, idx, idx_cap);
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
                                                           uint2* __restrict__ rk, uint32_t* __restrict__ pre, uint32_t* __restrict__ trank,
                                                           int32_t* __restrict__ idx, int64_t idx_cap) {
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
  const uint32_t j = s_prefix + ws[wid] + incl - n;
  if (c < n_chunks) {
    const uint32_t pb = chunk_prefix_bytes(__popc(w.x), __popc(w.y), __popc(w.z), __popc(w.w));
    rk[c] = make_uint2(j, pb);
    pre[c] = pb;
    if ((c & 7) == 0) trank[c >> 3] = j;
    if (c == n_chunks - 1) trank[(c >> 3) + 1] = j + n;      // the table's last entry: every set bit
  }
  write_chunk_indices(w, n, j, c, idx, idx_cap);           // whole warps (past the end: w = 0, n = 0)
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

// workers: the mask words two owners share, collected for their all-reduce and put back (scape_step_exchange)
__global__ void gather_words_kernel(const uint32_t* __restrict__ bits, const uint32_t* __restrict__ which, int n, uint32_t* __restrict__ out) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) out[i] = bits[which[i]];
}
__global__ void scatter_words_kernel(uint32_t* __restrict__ bits, const uint32_t* __restrict__ which, int n, const uint32_t* __restrict__ in) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) bits[which[i]] = in[i];
}

__global__ void fill_u32_kernel(uint32_t* p, int64_t n, uint32_t v) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) p[i] = v;
}

__global__ void iota_i32_kernel(int32_t* p, int64_t n, int32_t first) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) p[i] = first + (int32_t)i;
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

// ------------------------------------------------------------------------------------------
// Algorithm 2, parameter side (PAPER.md:222-242; Eq. 6, :207-211).  With a partitioned optimizer
// only the owner of a partition holds its updated parameters; the others bring their copies up to
// date from the owner's values on the mask the last update used (l.2-3) and decay the rest locally
// from their FP32 copy (l.4, "Use FP32 w to compute untransmitted params").
// ------------------------------------------------------------------------------------------
// l.2: out[j] = theta[idx[first + j]], j < count (ascending index order = the order of the sparse
// buffer); idx == nullptr: the mask is all ones and the payload is theta[first .. first + count).
// Four entries per thread in flight: the gather depends on the index load.
template <bool BF16>
__global__ void __launch_bounds__(256) param_pack_kernel(const float* __restrict__ theta, const int32_t* __restrict__ idx,
                                                        int64_t first, int64_t count, void* __restrict__ out) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t j0 = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; j0 < count; j0 += 4 * stride) {
    int64_t i[4]; float v[4]; bool ok[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int64_t j = j0 + u * stride;
      ok[u] = j < count;
      i[u] = ok[u] ? (idx ? (int64_t)__ldg(idx + first + j) : first + j) : 0;
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) v[u] = ok[u] ? __ldg(theta + i[u]) : 0.0f;
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      if (!ok[u]) continue;
      const int64_t j = j0 + u * stride;
      if (BF16) reinterpret_cast<__nv_bfloat16*>(out)[j] = __float2bfloat16_rn(v[u]);
      else reinterpret_cast<float*>(out)[j] = v[u];
    }
  }
}

__device__ __forceinline__ float payload_at(const void* __restrict__ p, bool bf16, int64_t j) {
  if (bf16) return __uint_as_float(((uint32_t)__ldg(reinterpret_cast<const uint16_t*>(p) + j)) << 16);
  return __ldg(reinterpret_cast<const float*>(p) + j);
}

// l.3-4 for one lane's 4 parameters of chunk c: on the mask w <- payload (packed position = rank128[c]
// + set bits before it), off the mask Alg. 1 l.17 with u = 0 (the owner's own arithmetic there:
// readings S13, S21); w^ = bf16(w).  mw / r0: the chunk's mask words and rank (all ones: unused).
template <bool BF16, bool HAT, bool ALLONES, bool GUARD>
__device__ __forceinline__ void param_apply_lane(float* __restrict__ w, uint16_t* __restrict__ w_hat, const void* __restrict__ payload,
                                                 int64_t N, int64_t c, int lane, const uint4 mw, const uint32_t r0, float (&v)[4],
                                                 float wd, float neg_lr) {
  const int64_t i0 = (c << 7) + ((int64_t)lane << 2);
  if (ALLONES) {
#pragma unroll
    for (int q = 0; q < 4; ++q) if (!GUARD || i0 + q < N) v[q] = payload_at(payload, BF16, i0 + q);
  } else {
    uint32_t mybits, jbase;
    lane_bits_from_words(mw, r0, lane, mybits, jbase);
    int64_t j = jbase;
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      const bool on = (mybits >> q) & 1u;
      const float dec = __fmaf_rn(neg_lr, __fmaf_rn(wd, v[q], 0.0f), v[q]);        // l.4 (Eq. 6 as l.17 with u = 0)
      v[q] = on ? payload_at(payload, BF16, j) : dec;                                // l.3
      j += on ? 1 : 0;
    }
  }
  store4_f32<GUARD>(w, i0, N, v);
  if (HAT) {
    if (!GUARD) {
      const uint32_t lo = (uint32_t)__bfloat16_as_ushort(__float2bfloat16_rn(v[0])) | ((uint32_t)__bfloat16_as_ushort(__float2bfloat16_rn(v[1])) << 16);
      const uint32_t hi = (uint32_t)__bfloat16_as_ushort(__float2bfloat16_rn(v[2])) | ((uint32_t)__bfloat16_as_ushort(__float2bfloat16_rn(v[3])) << 16);
      __stcs(reinterpret_cast<uint2*>(w_hat + i0), make_uint2(lo, hi));
    } else {
#pragma unroll
      for (int q = 0; q < 4; ++q) if (i0 + q < N) w_hat[i0 + q] = __bfloat16_as_ushort(__float2bfloat16_rn(v[q]));
    }
  }
}

// Streaming pass over the shard: reads w (4 B), writes w (4 B) and w^ (2 B) per parameter, plus the
// mask words, rank128 and the payload (k values).  HBM-bound; a warp takes kApplyChunks chunks per
// trip so that as many 128-bit loads per lane are in flight (10 bytes per parameter are too few
// for one: 2 per trip reached 84 % of the measured copy bandwidth).
constexpr int kApplyChunks = 4;
template <bool BF16, bool HAT, bool ALLONES>
__global__ void __launch_bounds__(256, 4) param_apply_kernel(float* __restrict__ w, uint16_t* __restrict__ w_hat,
                                                         const uint32_t* __restrict__ bits, const uint2* __restrict__ rank,
                                                         const void* __restrict__ payload, int64_t N, int64_t n_chunks,
                                                         float wd, float neg_lr) {
  const int lane = threadIdx.x & 31;
  const int64_t wpb = blockDim.x >> 5;
  const int64_t warp = (int64_t)blockIdx.x * wpb + (threadIdx.x >> 5);
  const int64_t nwarps = (int64_t)gridDim.x * wpb;
  const int64_t full = N >> 7;
  int64_t c = warp;
  for (; c + (kApplyChunks - 1) * nwarps < full; c += kApplyChunks * nwarps) {
    uint4 mw[kApplyChunks];
    uint32_t r0[kApplyChunks];
    float v[kApplyChunks][4];
#pragma unroll
    for (int u = 0; u < kApplyChunks; ++u) {
      mw[u] = make_uint4(0, 0, 0, 0); r0[u] = 0;
      if (!ALLONES) { mw[u] = __ldg(reinterpret_cast<const uint4*>(bits) + (c + u * nwarps)); r0[u] = __ldg(rank + (c + u * nwarps)).x; }
    }
#pragma unroll
    for (int u = 0; u < kApplyChunks; ++u)
      if (!ALLONES) load4_f32<false>(w, ((c + u * nwarps) << 7) + ((int64_t)lane << 2), N, v[u]);
#pragma unroll
    for (int u = 0; u < kApplyChunks; ++u)
      param_apply_lane<BF16, HAT, ALLONES, false>(w, w_hat, payload, N, c + u * nwarps, lane, mw[u], r0[u], v[u], wd, neg_lr);
  }
  for (; c < n_chunks; c += nwarps) {                        // the last trips, and the ragged last chunk
    uint4 ma = make_uint4(0, 0, 0, 0);
    uint32_t ra = 0;
    if (!ALLONES) { ma = __ldg(reinterpret_cast<const uint4*>(bits) + c); ra = __ldg(rank + c).x; }
    float va[4] = {0.0f, 0.0f, 0.0f, 0.0f};
    if (c < full) {
      if (!ALLONES) load4_f32<false>(w, (c << 7) + ((int64_t)lane << 2), N, va);
      param_apply_lane<BF16, HAT, ALLONES, false>(w, w_hat, payload, N, c, lane, ma, ra, va, wd, neg_lr);
    } else {
      if (!ALLONES) load4_f32<true>(w, (c << 7) + ((int64_t)lane << 2), N, va);
      param_apply_lane<BF16, HAT, ALLONES, true>(w, w_hat, payload, N, c, lane, ma, ra, va, wd, neg_lr);
    }
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
