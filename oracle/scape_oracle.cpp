// ORACLE — TEST INFRASTRUCTURE ONLY.
//
// Plain, slow, single-threaded CPU restatement of Algorithm 1 of SCAPE
// (arXiv 2607.01678) for ONE rank's partition with R simulated
// data-parallel replicas.  It exists so that tests can check the CUDA path against
// something a reader can compare with the paper by eye.  Only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// load it.  It shares no code with paper_2607_01678_b200/ (the product) and the
// product never calls it.
//
// Parity pins (tests/test_oracle_pins.py, all `-m "not gpu"`):
//   P1 top-k vs brute-force rank count      P2 packed + residual == m-tilde (bitwise)
//   P3 sparsity 0 == dense AdamS (Eq. 2)    P4 Eq. 3 reconstruction identity
//   P5 Eq. 4-6 off-mask behaviour           P6 telescoped error feedback (nothing lost)
//   P7 one-step mask delay                  P8 R = 1
//   P9 worked example tests/golden/p9_worked_example.json
//   P10 bias correction / learning-rate schedule == independent numpy Eq. 2 + PAPER.md:77 (dense)
//   P11 clip_grad: norm and factor vs numpy; no-op below the threshold; theta vs numpy (dense)
//   P12 per-layer refresh vs brute force per layer; exactly k_l per layer; one layer == flat
//   P13 an uncompressed layer is dense AdamS (Eq. 2) on its slice while the others are sparse
//   P14 sparsity schedule: mask counts follow the schedule with the one-step delay; P6 still holds
//   P15 workers: every layer's mask == brute force on ITS OWNER's |m-tilde|; the
//       two-level sum equals the flat mean (double, 1e-15); W = R with one owner == the plain step
//   P16 mask bit pack / unpack (oracle/scape_oracle.py, a plain loop) vs numpy packbits and an example
//   P17 bf16 round-to-nearest-even vs the torch CPU conversion, crafted ties, denormals, +-0
//   P18 Algorithm 2 parameter side: a non-owner's FP32 copy kept up by pack / all-gather / apply equals
//       the owner's theta of Algorithm 1 bit for bit, every step (fp32 payload); with a bf16 payload
//       the compute copy equals bf16(theta) on the mask; the mask of the exchange is the one the last
//       update used (any other mask breaks it)
//   P19 hand example tests/golden/p19_alg2_param_example.json;  P20 Eq. 6 literal vs l.17 with u = 0: <= 1 ulp
// Unpinned by the paper (decisions): S3 clip_grad off by default and,
// when switched on, the torch/Megatron rule; S4 bias correction off by default; S8 replica 0 owns
// the statistic; S9 flat top-k by default, per-layer top-k with uncompressed
// layers (:246, :279, :286) after set_layers; S19 the density warm-up schedule (:279) is the caller's.
//
// The algorithm is instantiated twice from the same template: T = float is the graded
// arithmetic (operation order pinned below);
// T = double exists only for the exact-arithmetic pins P3, P4, P6.
//
// Build: g++ -O2 -std=c++17 -ffp-contract=off -shared -fPIC   (see oracle/build.py)
// -ffp-contract=off matters: every rounding below is written out, the compiler must not
// fuse a*b+c on its own.

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <numeric>
#include <vector>

namespace {

// Sort key of the selection statistic abs(m-tilde) (Alg. 1 l.11; §IV-B,
// PAPER.md:182).  For finite IEEE numbers the unsigned bit pattern of |x| orders exactly
// like |x|; -0 and +0 get the same key.
template <class T> struct KeyOf;
template <> struct KeyOf<float> {
  using U = uint32_t;
  static U key(float x) { float a = std::fabs(x); U u; std::memcpy(&u, &a, sizeof u); return u; }
};
template <> struct KeyOf<double> {
  using U = uint64_t;
  static U key(double x) { double a = std::fabs(x); U u; std::memcpy(&u, &a, sizeof u); return u; }
};

template <class T>
struct Oracle {
  using U = typename KeyOf<T>::U;

  int64_t N = 0;
  int R = 0;
  int64_t k = 0;      // number selected per refresh: k = N - floor(sparsity * N)  (reading S6)
  int64_t t = 0;      // steps taken
  T beta1, beta2, eps, lr, wd;
  T c1, c2;           // 1 - beta1, 1 - beta2, evaluated in T
  double beta1_d, beta2_d;   // as given, for the bias-correction powers
  // Optional parts of Alg. 1 / Eq. 2 that the default configuration leaves out (readings S3, S4):
  bool bias_correction = false;   // m_t/(1-beta1^t), v_t/(1-beta2^t)
  double clip_max_norm = 0.0;     // l.14 clip_grad, 0 = off (PAPER.md:165; "gradient clip of 1", :279)
  double last_norm = 0.0;         // ||g^||_2 of the last step and the factor applied
  T last_coef = (T)1;

  // Per-layer refresh (PAPER.md:89 "per-layer style", :138 "number of layers in model L"): the
  // shard is cut into layers [off[l], off[l+1]); refresh_mask runs inside each layer with
  // k_l = n_l - floor(s * n_l); a layer with compress[l] == 0 is never sparsified (LayerNorm,
  // RMSNorm, bias: PAPER.md:246, :279, :286): all its entries are selected.  Empty = one layer.
  std::vector<int64_t> layer_off;
  std::vector<uint8_t> layer_compress;
  // Workers ("N workers", §IV-A :178 "each worker only computes a portion of the
  // top-k operations ... the new local masks from all workers are gathered"): the R replicas are
  // `workers` groups of R/workers consecutive replicas (one group = the gradient buffers of one
  // worker); layer l's statistic is the m-tilde of the FIRST replica of worker layer_owner[l]; the
  // mean of l.10 is taken the way an all-reduce over workers takes it: each worker sums its own
  // replicas in order, the workers' sums are added in worker order, one division by R.
  // workers = 1 (default) is the plain reading S8 / S14.
  int workers = 1;
  std::vector<int32_t> layer_owner;
  // Sparsity used by the NEXT refresh (density warm-up: "exponentially decrease
  // density d from 1 to 0.1 or 0.01"; the schedule itself is the caller's).
  double sparsity_now = 0.0;

  std::vector<T> m;                 // m_{t-1}, zero off the previous mask (Eq. 4)
  std::vector<std::vector<T>> e;    // e^r_{t-1}, one residual per replica (Alg. 1 l.2, :141)
  std::vector<uint8_t> cur;         // M_{t-1}, the mask used by the coming step (l.1: all ones)

  // What the last step produced (kept for inspection by tests).
  std::vector<int32_t> idx;             // ascending indices of the mask the step used
  std::vector<std::vector<T>> mt;       // m-tilde^r, all N entries (l.6)
  std::vector<std::vector<T>> b;        // packed payload b^r[j] = m-tilde^r[idx[j]] (l.9)
  std::vector<T> bbar;                  // mean payload (l.10)
  std::vector<T> ghat, v, u;            // l.13, l.15, l.16 on the mask, by position j

  Oracle(int64_t N_, int R_, double sparsity, double b1, double b2, double eps_, double lr_, double wd_)
      : N(N_), R(R_) {
    // Hyper-parameters are cast to T once; 1 - beta is evaluated in T.
    beta1 = (T)b1; beta2 = (T)b2; eps = (T)eps_; lr = (T)lr_; wd = (T)wd_;
    beta1_d = b1; beta2_d = b2;
    c1 = (T)1 - beta1;
    c2 = (T)1 - beta2;
    // Reading S6: k = N - floor(s*N) in IEEE double.
    k = N - (int64_t)std::floor(sparsity * (double)N);
    sparsity_now = sparsity;
    m.assign(N, (T)0);                                   // reading S5: m_0 = 0
    e.assign(R, std::vector<T>(N, (T)0));                // l.2: e_0 = 0
    cur.assign(N, 1);                                    // l.1: M_0 = 1
  }

  // refresh_mask (l.11): the k entries with the largest key; ties to the lower index (S7).
  // Written as the definition: stable sort of all indices by key, descending; take k.
  static std::vector<uint8_t> topk_mask(const T* x, int64_t n, int64_t kk) {
    std::vector<int64_t> order(n);
    std::iota(order.begin(), order.end(), (int64_t)0);
    std::stable_sort(order.begin(), order.end(), [&](int64_t a, int64_t c) {
      return KeyOf<T>::key(x[a]) > KeyOf<T>::key(x[c]);
    });
    std::vector<uint8_t> mask(n, 0);
    for (int64_t j = 0; j < kk; ++j) mask[order[j]] = 1;
    return mask;
  }

  static int64_t k_of(int64_t n, double sparsity) { return n - (int64_t)std::floor(sparsity * (double)n); }   // S6

  // l.11 with the per-layer reading: refresh_mask inside every layer, at the current sparsity,
  // from the statistic of the worker that owns the layer (worker 0 unless set_workers said otherwise).
  std::vector<uint8_t> refresh(const std::vector<std::vector<T>>& x) const {
    if (layer_off.empty()) return topk_mask(x[0].data(), N, k_of(N, sparsity_now));
    std::vector<uint8_t> mask(N, 0);
    const int Rl = R / workers;
    for (size_t l = 0; l + 1 < layer_off.size(); ++l) {
      const int64_t a = layer_off[l], n = layer_off[l + 1] - a;
      if (!layer_compress[l]) { std::fill(mask.begin() + a, mask.begin() + a + n, (uint8_t)1); continue; }
      const int owner = layer_owner.empty() ? 0 : layer_owner[l];
      std::vector<uint8_t> ml = topk_mask(x[owner * Rl].data() + a, n, k_of(n, sparsity_now));
      std::copy(ml.begin(), ml.end(), mask.begin() + a);
    }
    return mask;
  }

  void step(T* theta, const T* const* g) {
    t += 1;                                              // l.3
    // Indices of M_{t-1}, ascending.
    idx.clear();
    for (int64_t i = 0; i < N; ++i) if (cur[i]) idx.push_back((int32_t)i);
    const int64_t K = (int64_t)idx.size();

    // l.6: m-tilde^r = beta1 m_{t-1} + (1 - beta1) g^r + e^r_{t-1}
    mt.assign(R, std::vector<T>(N));
    for (int r = 0; r < R; ++r)
      for (int64_t i = 0; i < N; ++i) {
        T p = beta1 * m[i];
        mt[r][i] = std::fma(c1, g[r][i], p) + e[r][i];
      }

    // l.4 + l.9: b^r <- 0; b^r[M_{t-1}] <- m-tilde^r[M_{t-1}]  (stored packed, by position j)
    b.assign(R, std::vector<T>(K));
    for (int r = 0; r < R; ++r)
      for (int64_t j = 0; j < K; ++j) b[r][j] = mt[r][idx[j]];

    // l.7-8: e^r[not M_{t-1}] <- m-tilde^r ; e^r[M_{t-1}] <- 0
    for (int r = 0; r < R; ++r)
      for (int64_t i = 0; i < N; ++i) e[r][i] = cur[i] ? (T)0 : mt[r][i];

    // l.11: M_t <- refresh_mask(density, abs(m-tilde)) from the owner's (replica 0) statistic,
    // over all N positions (readings S8, S11).  Used from the next step on (§IV-A, :178).
    // With layers set: the same inside every layer.
    std::vector<uint8_t> next = refresh(mt);

    // l.10, l.12-17 on the mask.
    std::vector<T> m_new(N, (T)0);                       // l.12 / Eq. 4: zero off the mask
    bbar.assign(K, (T)0); ghat.assign(K, (T)0); v.assign(K, (T)0); u.assign(K, (T)0);
    for (int64_t j = 0; j < K; ++j) {
      const int64_t i = idx[j];
      const int Rl = R / workers;                        // replicas per worker (R when workers = 1)
      T s = (T)0;
      for (int w = 0; w < workers; ++w) {                // l.10: all-reduce = sum of the workers' sums
        T sw = b[w * Rl][j];                             //   one worker: its replicas, r ascending
        for (int r = 1; r < Rl; ++r) sw = sw + b[w * Rl + r][j];
        s = w == 0 ? sw : s + sw;
      }
      T bb = s / (T)R;
      T p = beta1 * m[i];
      bbar[j] = bb;
      ghat[j] = (bb - p) / c1;                           // l.13 (Eq. 3, :188)
    }
    // l.14 clip_grad(b-bar): global-norm clip of the reconstructed gradient over the mask.
    // The paper does not define it; this is the usual rule (torch / Megatron clip_grad_norm):
    // coef = max_norm / (||g^||_2 + 1e-6), applied only when coef < 1.  The norm is accumulated in
    // double, in index order.
    T coef = (T)1;
    {
      double ss = 0.0;
      for (int64_t j = 0; j < K; ++j) ss += (double)ghat[j] * (double)ghat[j];
      last_norm = std::sqrt(ss);
      if (clip_max_norm > 0.0) {
        const double cc = clip_max_norm / (last_norm + 1e-6);
        if (cc < 1.0) coef = (T)cc;
      }
      last_coef = coef;
    }
    // Bias correction, off by default (reading S4): factors 1/(1-beta^t) evaluated in
    // double from the step number, cast to T once.
    T bc1 = (T)1, bc2 = (T)1;
    if (bias_correction) {
      bc1 = (T)(1.0 / (1.0 - std::pow(beta1_d, (double)t)));
      bc2 = (T)(1.0 / (1.0 - std::pow(beta2_d, (double)t)));
    }
    for (int64_t j = 0; j < K; ++j) {
      const int64_t i = idx[j];
      const T bb = bbar[j];
      T gh = ghat[j];
      if (clip_max_norm > 0.0) gh = gh * coef;           // l.14
      T vv = std::fma(c2, gh * gh, beta2 * (m[i] * m[i]));   // l.15
      T uu = (bb * bc1) / (std::sqrt(vv * bc2) + eps);   // l.16 with m_t = bbar (l.12)
      T w = std::fma(wd, theta[i], uu);                  // l.17
      theta[i] = std::fma(-lr, w, theta[i]);
      m_new[i] = bb;                                     // l.12
      ghat[j] = gh; v[j] = vv; u[j] = uu;
    }
    // Off the mask: u = 0 (Eq. 5, :202), so l.17 is pure weight decay (Eq. 6, :207-211).
    for (int64_t i = 0; i < N; ++i) {
      if (cur[i]) continue;
      T uu = (T)0;
      T w = std::fma(wd, theta[i], uu);
      theta[i] = std::fma(-lr, w, theta[i]);
    }
    m.swap(m_new);
    cur.swap(next);                                      // the delay: M_t is used at step t+1
  }
};

template <class T> void copy_out(const std::vector<T>& v, T* dst) {
  if (!v.empty()) std::memcpy(dst, v.data(), v.size() * sizeof(T));
}

}  // namespace

#define ORACLE_API(SUF, T)                                                                          \
  extern "C" void* oracle_create_##SUF(int64_t N, int R, double sparsity, double b1, double b2,     \
                                       double eps, double lr, double wd) {                          \
    if (N <= 0 || N >= (int64_t)1 << 31 || R < 1 || !(sparsity >= 0.0 && sparsity < 1.0))           \
      return nullptr;                                                                               \
    return new Oracle<T>(N, R, sparsity, b1, b2, eps, lr, wd);                                      \
  }                                                                                                 \
  extern "C" void oracle_destroy_##SUF(void* h) { delete (Oracle<T>*)h; }                           \
  extern "C" void oracle_step_##SUF(void* h, T* theta, const T* const* grads) {                     \
    ((Oracle<T>*)h)->step(theta, grads);                                                            \
  }                                                                                                 \
  extern "C" int64_t oracle_k_##SUF(void* h) { return ((Oracle<T>*)h)->k; }                         \
  extern "C" int64_t oracle_t_##SUF(void* h) { return ((Oracle<T>*)h)->t; }                         \
  extern "C" int64_t oracle_K_last_##SUF(void* h) { return (int64_t)((Oracle<T>*)h)->idx.size(); }  \
  extern "C" void oracle_get_m_##SUF(void* h, T* dst) { copy_out(((Oracle<T>*)h)->m, dst); }        \
  extern "C" void oracle_set_m_##SUF(void* h, const T* src) {                                       \
    auto* o = (Oracle<T>*)h; std::memcpy(o->m.data(), src, o->N * sizeof(T));                       \
  }                                                                                                 \
  extern "C" void oracle_get_e_##SUF(void* h, int r, T* dst) { copy_out(((Oracle<T>*)h)->e[r], dst); } \
  extern "C" void oracle_set_e_##SUF(void* h, int r, const T* src) {                                \
    auto* o = (Oracle<T>*)h; std::memcpy(o->e[r].data(), src, o->N * sizeof(T));                    \
  }                                                                                                 \
  extern "C" void oracle_get_mask_##SUF(void* h, uint8_t* dst) {                                    \
    copy_out(((Oracle<T>*)h)->cur, dst);                                                            \
  }                                                                                                 \
  extern "C" void oracle_set_mask_##SUF(void* h, const uint8_t* src) {                              \
    auto* o = (Oracle<T>*)h; std::memcpy(o->cur.data(), src, o->N);                                 \
  }                                                                                                 \
  extern "C" void oracle_set_t_##SUF(void* h, int64_t t) { ((Oracle<T>*)h)->t = t; }                \
  extern "C" int oracle_set_layers_##SUF(void* h, int L, const int64_t* off, const uint8_t* compress) { \
    auto* o = (Oracle<T>*)h;                                                                        \
    if (L < 1 || off[0] != 0 || off[L] != o->N) return -1;                                          \
    for (int l = 0; l < L; ++l) if (off[l + 1] <= off[l]) return -1;                                \
    o->layer_off.assign(off, off + L + 1); o->layer_compress.assign(compress, compress + L);        \
    o->layer_owner.clear();                                                                         \
    return 0;                                                                                       \
  }                                                                                                 \
  extern "C" int oracle_set_workers_##SUF(void* h, int W, const int32_t* owner) {                  \
    auto* o = (Oracle<T>*)h;                                                                        \
    if (W < 1 || o->R % W != 0) return -1;                                                          \
    const size_t L = o->layer_off.empty() ? 0 : o->layer_off.size() - 1;                            \
    if (owner) { if (L == 0) return -1; for (size_t l = 0; l < L; ++l) if (owner[l] < 0 || owner[l] >= W) return -1; } \
    o->workers = W;                                                                                 \
    if (owner) o->layer_owner.assign(owner, owner + L); else o->layer_owner.clear();                \
    return 0;                                                                                       \
  }                                                                                                 \
  extern "C" int oracle_set_sparsity_##SUF(void* h, double s) {                                     \
    if (!(s >= 0.0 && s < 1.0)) return -1;                                                          \
    auto* o = (Oracle<T>*)h; o->sparsity_now = s; o->k = Oracle<T>::k_of(o->N, s); return 0;        \
  }                                                                                                 \
  extern "C" void oracle_set_lr_##SUF(void* h, double lr) { ((Oracle<T>*)h)->lr = (T)lr; }         \
  extern "C" void oracle_set_bias_correction_##SUF(void* h, int on) { ((Oracle<T>*)h)->bias_correction = on != 0; } \
  extern "C" void oracle_set_clip_grad_##SUF(void* h, double c) { ((Oracle<T>*)h)->clip_max_norm = c; } \
  extern "C" double oracle_last_norm_##SUF(void* h) { return ((Oracle<T>*)h)->last_norm; }          \
  extern "C" double oracle_last_coef_##SUF(void* h) { return (double)((Oracle<T>*)h)->last_coef; }                \
  extern "C" void oracle_get_idx_##SUF(void* h, int32_t* dst) { copy_out(((Oracle<T>*)h)->idx, dst); } \
  extern "C" void oracle_get_mt_##SUF(void* h, int r, T* dst) { copy_out(((Oracle<T>*)h)->mt[r], dst); } \
  extern "C" void oracle_get_b_##SUF(void* h, int r, T* dst) { copy_out(((Oracle<T>*)h)->b[r], dst); } \
  extern "C" void oracle_get_bbar_##SUF(void* h, T* dst) { copy_out(((Oracle<T>*)h)->bbar, dst); }  \
  extern "C" void oracle_get_ghat_##SUF(void* h, T* dst) { copy_out(((Oracle<T>*)h)->ghat, dst); }  \
  extern "C" void oracle_get_v_##SUF(void* h, T* dst) { copy_out(((Oracle<T>*)h)->v, dst); }        \
  extern "C" void oracle_get_u_##SUF(void* h, T* dst) { copy_out(((Oracle<T>*)h)->u, dst); }        \
  extern "C" void oracle_topk_##SUF(const T* x, int64_t n, int64_t kk, uint8_t* mask) {             \
    auto mk = Oracle<T>::topk_mask(x, n, kk); std::memcpy(mask, mk.data(), (size_t)n);              \
  }

ORACLE_API(f32, float)
ORACLE_API(f64, double)

// ---------------------------------------------------------------------------------------------
// Algorithm 2, parameter side (PAPER.md:222-242; Eq. 6, :207-211; "Use FP32 w to compute
// untransmitted params", :231-232).  With a partitioned (distributed) optimizer only the OWNER of a
// partition holds its updated parameters w'.  Every other worker keeps a full FP32 copy w and the
// compute copy w^ (BF16 parameters), and brings both up to date from
//   l.2  w~ <- w'[M]                      the owner's updated parameters on the mask, packed in
//                                         ascending index order (fp32, or rounded to bf16: RNE)
//   l.3  w^[M] <- AllGather(w~)           (the all-gather itself is the caller's)
//   l.4  w^[not M] <- (1 - eta lambda) w^[not M], computed from the FP32 copy w
// where M is the mask the last update used (Eq. 6 is about theta_{t+1}[not M_{t-1}]; DESIGN.md
// reading S22).  Reading S21: the FP32 copy is updated in place, w[M] <- payload, w[not M] by
// Alg. 1 l.17 with u = 0 -- fma(-eta, lambda*w, w), the arithmetic the owner itself applies off the
// mask (reading S13) -- so that with an fp32 payload the copy equals the owner's theta to the bit;
// w^ = bf16(w) everywhere.  form = 1 computes Eq. 6 literally, (1 - eta*lambda) * w, for pin P20.
// ---------------------------------------------------------------------------------------------
namespace {

// float -> bfloat16, round to nearest, ties to even, written out from the definition: keep the upper
// 16 bits; the dropped 16 bits are compared with one half (0x8000); above -> up, below -> down,
// exactly half -> towards the even kept value.  NaN keeps its sign and gets a quiet payload.
uint16_t bf16_rne(float x) {
  uint32_t u;
  std::memcpy(&u, &x, sizeof u);
  if ((u & 0x7F800000u) == 0x7F800000u && (u & 0x007FFFFFu) != 0u) return (uint16_t)((u >> 16) | 0x0040u);   // NaN
  const uint32_t kept = u >> 16, dropped = u & 0xFFFFu;
  uint32_t r = kept;
  if (dropped > 0x8000u) r = kept + 1u;
  else if (dropped == 0x8000u) r = kept + (kept & 1u);
  return (uint16_t)r;          // a carry out of the mantissa moves to the next exponent (or to inf): correct by construction
}

float bf16_widen(uint16_t b) {
  const uint32_t u = (uint32_t)b << 16;
  float x;
  std::memcpy(&x, &u, sizeof x);
  return x;
}

}  // namespace

extern "C" uint16_t oracle_bf16_rne(float x) { return bf16_rne(x); }
extern "C" float oracle_bf16_widen(uint16_t b) { return bf16_widen(b); }
extern "C" void oracle_bf16_rne_array(const float* x, int64_t n, uint16_t* out) { for (int64_t i = 0; i < n; ++i) out[i] = bf16_rne(x[i]); }

// l.2: out[j] = w_local[i_j], i_0 < i_1 < ... the positions with mask[i] != 0.  Returns the count.
// out_f32 or out_bf16 (exactly one non-null).
extern "C" int64_t oracle_param_pack(const float* w_local, const uint8_t* mask, int64_t N, float* out_f32, uint16_t* out_bf16) {
  int64_t j = 0;
  for (int64_t i = 0; i < N; ++i) {
    if (!mask[i]) continue;
    if (out_f32) out_f32[j] = w_local[i];
    if (out_bf16) out_bf16[j] = bf16_rne(w_local[i]);
    ++j;
  }
  return j;
}

// l.3-4 on a non-owner: w [N] FP32 copy, updated in place; w_hat [N] bf16 compute copy (may be null);
// payload in ascending index order of the mask, fp32 or bf16 (exactly one non-null).
extern "C" void oracle_param_apply(float* w, uint16_t* w_hat, const uint8_t* mask, int64_t N, const float* payload_f32,
                                   const uint16_t* payload_bf16, double lr_d, double wd_d, int form) {
  const float lr = (float)lr_d, wd = (float)wd_d;           // cast once, like Alg. 1's hyper-parameters
  int64_t j = 0;
  for (int64_t i = 0; i < N; ++i) {
    if (mask[i]) {                                           // l.3
      w[i] = payload_f32 ? payload_f32[j] : bf16_widen(payload_bf16[j]);
      ++j;
    } else if (form == 0) {                                  // l.4 as Alg. 1 l.17 with u = 0 (S13, S21)
      const float d = std::fma(wd, w[i], 0.0f);
      w[i] = std::fma(-lr, d, w[i]);
    } else {                                                 // l.4 / Eq. 6 literally
      const float f = 1.0f - lr * wd;
      w[i] = f * w[i];
    }
    if (w_hat) w_hat[i] = bf16_rne(w[i]);
  }
}
