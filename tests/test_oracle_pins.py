"""Pins of the CPU oracle against what the paper and the mathematics fix (CPU only).

Each test names the pin (P1..P9, SURVEY.md §8(c)-5 / DESIGN.md §Oracle pins) and the passage of
PAPER.md it rests on.  None of the expected values comes from oracle/ or from the CUDA path:
they are brute force, closed forms, invariants, independent numpy restatements of Eq. 2, or
the hand-derived golden fixture.
"""
import json
import os

import numpy as np
import pytest

from oracle.scape_oracle import ScapeOracle, topk_mask

HERE = os.path.dirname(os.path.abspath(__file__))
HYP = dict(beta1=0.9, beta2=0.95, eps=1e-8, lr=1e-3, wd=0.1)


def make_grads(rng, N, R, T, dtype=np.float32, rho=0.9):
    """AR(1) signal + per-replica noise, as in BASELINE.json config 1."""
    out, a = [], None
    for _ in range(T):
        xi = rng.standard_normal(N)
        a = xi if a is None else rho * a + np.sqrt(1 - rho * rho) * xi
        out.append([(1e-3 * (a + rng.standard_normal(N))).astype(dtype) for _ in range(R)])
    return out


def ulp32(x):
    return np.spacing(np.abs(np.asarray(x, dtype=np.float32)))


# ------------------------------------------------------------------------------------ P1
def brute_force_topk(x, k):
    """Definition (reading S7): rank_i = #{j : |x_j| > |x_i| or (|x_j| == |x_i| and j < i)};
    selected iff rank_i < k.  O(n^2), written without any sort."""
    a = np.abs(x)
    n = len(x)
    mask = np.zeros(n, dtype=np.uint8)
    for i in range(n):
        rank = 0
        for j in range(n):
            if a[j] > a[i] or (a[j] == a[i] and j < i):
                rank += 1
        mask[i] = 1 if rank < k else 0
    return mask


CRAFTED = {
    "all_equal": np.full(17, 0.25, np.float32),
    "pm_pairs": np.array([1, -1, 2, -2, 3, -3, 0.5, -0.5], np.float32),
    "zeros": np.zeros(9, np.float32),
    "signed_zeros": np.array([0.0, -0.0, 0.0, -0.0, 1.0], np.float32),
    "dups_straddle": np.array([5, 3, 3, 3, 3, 1, 3, 0, 3], np.float32),
    "denormals": np.array([1e-45, -3e-45, 2e-45, 0, 1e-38, -1e-45], np.float32),
    "descending": np.arange(20, 0, -1).astype(np.float32),
    "ascending": np.arange(1, 21).astype(np.float32),
}


@pytest.mark.parametrize("name", sorted(CRAFTED))
def test_p1_topk_crafted_vs_brute_force(name):
    x = CRAFTED[name]
    for k in range(1, len(x) + 1):
        got = topk_mask(x, k)
        assert got.sum() == k
        np.testing.assert_array_equal(got, brute_force_topk(x, k), err_msg=f"{name} k={k}")


@pytest.mark.parametrize("seed", range(6))
def test_p1_topk_random_vs_brute_force(seed):
    rng = np.random.default_rng(seed)
    n = int(rng.integers(2, 65))
    # few distinct magnitudes -> many ties
    x = (rng.integers(-4, 5, n) * 0.125).astype(np.float32)
    y = rng.standard_normal(n).astype(np.float32)
    for v in (x, y, y.astype(np.float64)):
        for k in {1, max(1, n // 10), n // 2 + 1, n}:
            np.testing.assert_array_equal(topk_mask(v, k), brute_force_topk(v, k))


def test_exactly_k_selected_and_k_rule():
    # Reading S6: k = N - floor(s N) in IEEE double.
    for N, s in [(1 << 20, 0.9), (1000, 0.99), (1000, 0.999), (7, 0.5), (354501632 // 1000, 0.99)]:
        o = ScapeOracle(N, 1, s, **HYP)
        assert o.k == N - int(np.floor(s * N))
    o = ScapeOracle(1 << 20, 2, 0.9, **HYP)
    assert o.k == 104858
    rng = np.random.default_rng(1)
    N, R = 4096, 2
    o = ScapeOracle(N, R, 0.9, **HYP)
    th = rng.standard_normal(N).astype(np.float32)
    for g in make_grads(rng, N, R, 4):
        o.step(th, g)
        mk = o.mask()
        assert mk.sum() == o.k
        idx = np.nonzero(mk)[0]
        assert np.all(np.diff(idx) > 0) and idx[-1] < N


def test_create_rejects_bad_arguments():
    for bad in [dict(N=0), dict(N=1 << 31), dict(R=0), dict(s=1.0), dict(s=-0.1), dict(s=float("nan"))]:
        args = dict(N=16, R=1, s=0.5)
        args.update(bad)
        with pytest.raises(ValueError):
            ScapeOracle(args["N"], args["R"], args["s"], **HYP)


# ------------------------------------------------------------------------------------ P2
def test_p2_packed_plus_residual_is_mtilde_bitwise():
    """'packed values plus residual equal the pre-mask quantity' (Alg. 1 l.7-9)."""
    rng = np.random.default_rng(2)
    N, R = 5000, 3
    o = ScapeOracle(N, R, 0.9, **HYP)
    th = (0.02 * rng.standard_normal(N)).astype(np.float32)
    for g in make_grads(rng, N, R, 5):
        o.step(th, g)
        idx = o.idx()
        on = np.zeros(N, bool)
        on[idx] = True
        for r in range(R):
            scat = np.zeros(N, np.float32)
            scat[idx] = o.b(r)
            e, mt = o.e(r), o.mt(r)
            # one of the two terms is exactly zero at every position
            assert np.all(e[on] == 0) and np.all(scat[~on] == 0)
            total = scat + e
            assert np.array_equal(total.view(np.uint32) & 0x7FFFFFFF, mt.view(np.uint32) & 0x7FFFFFFF)
            nz = mt != 0
            assert np.array_equal(total.view(np.uint32)[nz], mt.view(np.uint32)[nz])


# ------------------------------------------------------------------------------------ P3
def dense_adams_f64(theta, m, gbar, beta1, beta2, eps, lr, wd):
    """Eq. 2, written independently of the oracle, no bias correction (S4)."""
    m_new = beta1 * m + (1 - beta1) * gbar
    v = beta2 * m * m + (1 - beta2) * gbar * gbar
    theta_new = theta - lr * (m_new / (np.sqrt(v) + eps) + wd * theta)
    return theta_new, m_new


def test_p3_sparsity_zero_is_dense_adams_double():
    rng = np.random.default_rng(3)
    N, R, T = 3000, 4, 6
    o = ScapeOracle(N, R, 0.0, dtype=np.float64, **HYP)
    assert o.k == N
    th = 0.02 * rng.standard_normal(N)
    th_ref, m_ref = th.copy(), np.zeros(N)
    for g in make_grads(rng, N, R, T, dtype=np.float64):
        o.step(th, g)
        gbar = sum(g) / R
        th_ref, m_ref = dense_adams_f64(th_ref, m_ref, gbar, **HYP)
        assert o.K_last == N and o.mask().all()
        for r in range(R):
            assert not o.e(r).any()
        np.testing.assert_allclose(o.m(), m_ref, rtol=1e-12, atol=1e-300)
        np.testing.assert_allclose(th, th_ref, rtol=1e-12, atol=1e-300)


def test_p3_sparsity_zero_is_dense_adams_fp32_loose():
    """fp32: l.13 re-derives g-bar through a cancellation, so not bitwise; 1e-5 on theta."""
    rng = np.random.default_rng(4)
    N, R, T = 3000, 2, 6
    o = ScapeOracle(N, R, 0.0, **HYP)
    th = (0.02 * rng.standard_normal(N)).astype(np.float32)
    th_ref, m_ref = th.astype(np.float64), np.zeros(N)
    for g in make_grads(rng, N, R, T):
        o.step(th, g)
        gbar = sum(x.astype(np.float64) for x in g) / R
        th_ref, m_ref = dense_adams_f64(th_ref, m_ref, gbar, **HYP)
    np.testing.assert_allclose(th, th_ref, rtol=1e-5, atol=1e-9)
    np.testing.assert_allclose(o.m(), m_ref, rtol=1e-5, atol=1e-9)   # |m| ~ 1e-3; near-zero entries cancel


# ------------------------------------------------------------------------------------ P4
def test_p4_eq3_reconstruction_identity_double():
    """Eq. 3 with l.6: (b-bar - beta1 m)/(1-beta1) = g-bar + e-bar/(1-beta1) (S2)."""
    rng = np.random.default_rng(5)
    N, R, T = 2000, 3, 6
    o = ScapeOracle(N, R, 0.9, dtype=np.float64, **HYP)
    th = 0.02 * rng.standard_normal(N)
    for g in make_grads(rng, N, R, T, dtype=np.float64):
        e_prev = [o.e(r) for r in range(R)]
        o.step(th, g)
        idx = o.idx()
        gbar = sum(g) / R
        ebar = sum(e_prev) / R
        want = gbar[idx] + ebar[idx] / (1 - HYP["beta1"])
        np.testing.assert_allclose(o.ghat(), want, rtol=1e-9, atol=1e-15)
    assert o.K_last == o.k      # after step 1 the mask has k entries


# ------------------------------------------------------------------------------------ P5
def test_p5_off_mask_eq4_5_6():
    rng = np.random.default_rng(6)
    N, R, T = 4000, 2, 8
    o = ScapeOracle(N, R, 0.99, **HYP)
    th = (0.02 * rng.standard_normal(N)).astype(np.float32)
    th0 = th.copy()
    ever = np.zeros(N, bool)
    decay = np.float32(1.0) - np.float32(HYP["lr"]) * np.float32(HYP["wd"])
    for g in make_grads(rng, N, R, T):
        before = th.copy()
        o.step(th, g)
        on = np.zeros(N, bool)
        on[o.idx()] = True
        ever |= on
        assert not o.m()[~on].any()                                   # Eq. 4
        want = before[~on] * decay                                   # Eq. 6
        assert np.all(np.abs(th[~on] - want) <= 2 * ulp32(want))     # l.17 form vs Eq. 6: <= ~1 ulp
    # the first step is dense (M_0 = 1), so "never selected" is judged from step 2 on
    o2 = ScapeOracle(N, R, 0.99, **HYP)
    th = th0.copy()
    gs = make_grads(np.random.default_rng(7), N, R, T)
    o2.step(th, gs[0])
    th1 = th.copy()
    never = np.ones(N, bool)
    for g in gs[1:]:
        o2.step(th, g)
        never[o2.idx()] = False
    want = th1[never].astype(np.float64) * (1 - HYP["lr"] * HYP["wd"]) ** (T - 1)
    assert never.sum() > N // 2
    assert np.all(np.abs(th[never] - want) <= (T + 1) * ulp32(want))


# ------------------------------------------------------------------------------------ P6
def test_p6_telescoped_error_feedback_double():
    """(1-b1) sum_{t<=T} gbar_t = ebar_T + m_T + (1-b1) sum_{t<T} m_t  (DESIGN.md §Oracle pins)."""
    rng = np.random.default_rng(8)
    N, R, T = 1500, 3, 12
    o = ScapeOracle(N, R, 0.95, dtype=np.float64, **HYP)
    th = 0.02 * rng.standard_normal(N)
    c1 = 1 - HYP["beta1"]
    sum_g, sum_m_before = np.zeros(N), np.zeros(N)
    for g in make_grads(rng, N, R, T, dtype=np.float64):
        sum_m_before += o.m()          # adds m_{t-1}; m_0 = 0
        o.step(th, g)
        sum_g += sum(g) / R
        ebar = sum(o.e(r) for r in range(R)) / R
        lhs = c1 * sum_g
        rhs = ebar + o.m() + c1 * sum_m_before
        np.testing.assert_allclose(lhs, rhs, rtol=1e-10, atol=1e-14)


# ------------------------------------------------------------------------------------ P7
def test_p7_mask_is_used_one_step_late():
    rng = np.random.default_rng(9)
    N, R = 2048, 2
    o = ScapeOracle(N, R, 0.9, **HYP)
    th = (0.02 * rng.standard_normal(N)).astype(np.float32)
    prev_next = None
    for t, g in enumerate(make_grads(rng, N, R, 5), 1):
        o.step(th, g)
        if t == 1:
            np.testing.assert_array_equal(o.idx(), np.arange(N, dtype=np.int32))   # M_0 = 1
        else:
            np.testing.assert_array_equal(o.idx(), np.nonzero(prev_next)[0].astype(np.int32))
        # the refreshed mask is the top-k of THIS step's |m-tilde^0| over all positions (l.11)
        np.testing.assert_array_equal(o.mask(), brute_force_topk_fast(o.mt(0), o.k))
        prev_next = o.mask()


def brute_force_topk_fast(x, k):
    """Same definition as brute_force_topk, via lexsort on (index, -|x|) — still independent of
    the oracle's stable_sort; used where n is too large for the O(n^2) loop."""
    order = np.lexsort((np.arange(len(x)), -np.abs(x.astype(np.float64))))
    mask = np.zeros(len(x), np.uint8)
    mask[order[:k]] = 1
    return mask


def test_brute_force_variants_agree():
    rng = np.random.default_rng(10)
    x = (rng.integers(-3, 4, 50) * 0.5).astype(np.float32)
    for k in (1, 7, 25, 50):
        np.testing.assert_array_equal(brute_force_topk(x, k), brute_force_topk_fast(x, k))


# ------------------------------------------------------------------------------------ P8
def test_p8_single_replica():
    rng = np.random.default_rng(11)
    N = 3000
    o = ScapeOracle(N, 1, 0.9, **HYP)
    od = ScapeOracle(N, 1, 0.9, dtype=np.float64, **HYP)
    th = (0.02 * rng.standard_normal(N)).astype(np.float32)
    thd = th.astype(np.float64)
    for g in make_grads(rng, N, 1, 5):
        e_prev = od.e(0)
        o.step(th, g)
        od.step(thd, [g[0].astype(np.float64)])
        assert np.array_equal(o.bbar().view(np.uint32), o.b(0).view(np.uint32))   # b-bar = b^0 bitwise
        idx = od.idx()
        want = g[0].astype(np.float64)[idx] + e_prev[idx] / (1 - HYP["beta1"])
        np.testing.assert_allclose(od.ghat(), want, rtol=1e-9, atol=1e-15)


# ------------------------------------------------------------------------------------ P9
def test_p9_worked_example_golden():
    with open(os.path.join(HERE, "golden", "p9_worked_example.json")) as f:
        G = json.load(f)
    o = ScapeOracle(G["N"], G["R"], G["sparsity"], G["beta1"], G["beta2"], G["eps"], G["lr"], G["wd"])
    assert o.k == G["k"]
    th = np.array(G["theta0"], np.float32)
    sc = np.float32(G["grad_scale"])
    for s in G["steps"]:
        g = [np.array(s["g0"], np.float32) * sc, np.array(s["g1"], np.float32) * sc]
        o.step(th, g)
        np.testing.assert_array_equal(o.idx(), np.array(s["cur"], np.int32))
        np.testing.assert_array_equal(np.nonzero(o.mask())[0], np.array(s["next"]))
        # exact (dyadic) quantities
        for r, key in ((0, "mt0"), (1, "mt1")):
            np.testing.assert_array_equal(o.mt(r), np.array(s[key], np.float32))
        for r, key in ((0, "b0"), (1, "b1")):
            np.testing.assert_array_equal(o.b(r), np.array(s[key], np.float32))
        for r, key in ((0, "e0_after"), (1, "e1_after")):
            np.testing.assert_array_equal(o.e(r), np.array(s[key], np.float32))
        np.testing.assert_array_equal(o.m(), np.array(s["m_after"], np.float32))
        K = len(s["cur"])
        take = (lambda a: np.array(a, np.float32)[np.array(s["cur"])]) if len(s["ghat"]) == G["N"] and K == G["N"] \
            else (lambda a: np.array(a, np.float32))
        np.testing.assert_array_equal(o.ghat(), take(s["ghat"]))
        np.testing.assert_array_equal(o.v(), take(s["v"]))
        # non-dyadic
        np.testing.assert_allclose(o.u(), take(s["u"]), rtol=1e-6, atol=0)
        np.testing.assert_allclose(th, np.array(s["theta_after"], np.float32), rtol=1e-6, atol=0)


# ------------------------------------------------------------------------- f32 vs f64 sanity
def test_f32_and_f64_instantiations_track_each_other():
    rng = np.random.default_rng(12)
    N, R = 2000, 2
    o32 = ScapeOracle(N, R, 0.9, **HYP)
    o64 = ScapeOracle(N, R, 0.9, dtype=np.float64, **HYP)
    th32 = (0.02 * rng.standard_normal(N)).astype(np.float32)
    th64 = th32.astype(np.float64)
    for g in make_grads(rng, N, R, 3):
        o32.step(th32, g)
        o64.step(th64, [x.astype(np.float64) for x in g])
    np.testing.assert_allclose(th32, th64, rtol=2e-4, atol=1e-7)


# ------------------------------------------------------------------------------------ P10
def dense_adams_full_f64(theta, m, gbar, t, beta1, beta2, eps, lr, wd, bias_correction, clip):
    """Eq. 2 + bias correction + global-norm clip of the gradient (Alg. 1 l.14 at
    density 1, where g-hat = g-bar), written independently of the oracle."""
    g = gbar
    norm = float(np.sqrt(np.sum(g * g)))
    coef = 1.0
    if clip > 0 and clip / (norm + 1e-6) < 1.0:
        coef = clip / (norm + 1e-6)
    g = g * coef if clip > 0 else g
    m_new = beta1 * m + (1 - beta1) * gbar          # l.12: the first moment is NOT clipped (clip follows it)
    v = beta2 * m * m + (1 - beta2) * g * g
    if bias_correction:
        mhat, vhat = m_new / (1 - beta1 ** t), v / (1 - beta2 ** t)
    else:
        mhat, vhat = m_new, v
    return theta - lr * (mhat / (np.sqrt(vhat) + eps) + wd * theta), m_new, norm, coef


@pytest.mark.parametrize("bc,clip", [(True, 0.0), (False, 0.05), (True, 0.05), (False, 1e9)])
def test_p10_p11_bias_correction_clip_and_lr_schedule_dense_double(bc, clip):
    rng = np.random.default_rng(13)
    N, R, T = 2500, 3, 7
    o = ScapeOracle(N, R, 0.0, dtype=np.float64, **HYP)
    o.set_bias_correction(bc)
    o.set_clip_grad(clip)
    th = 0.02 * rng.standard_normal(N)
    th_ref, m_ref = th.copy(), np.zeros(N)
    clipped_once = False
    for t, g in enumerate(make_grads(rng, N, R, T, dtype=np.float64), 1):
        lr = HYP["lr"] * (0.5 + 0.1 * t)             # a schedule
        o.set_lr(lr)
        o.step(th, g)
        gbar = sum(g) / R
        hyp = dict(HYP, lr=lr)
        th_ref, m_ref, norm, coef = dense_adams_full_f64(th_ref, m_ref, gbar, t, bias_correction=bc, clip=clip, **hyp)
        np.testing.assert_allclose(o.last_norm(), norm, rtol=1e-9)       # g-hat = g-bar up to the l.13 round trip
        np.testing.assert_allclose(o.last_coef(), coef, rtol=1e-9)
        clipped_once |= coef < 1.0
        np.testing.assert_allclose(o.m(), m_ref, rtol=1e-12, atol=1e-300)
        np.testing.assert_allclose(th, th_ref, rtol=1e-9, atol=1e-300)
    assert clipped_once == (0 < clip < 1)             # the 0.05 threshold does bite, 1e9 never does


def test_p11_clip_below_threshold_is_bitwise_noop_fp32():
    rng = np.random.default_rng(14)
    N, R = 3000, 2
    a, b = ScapeOracle(N, R, 0.9, **HYP), ScapeOracle(N, R, 0.9, **HYP)
    b.set_clip_grad(1e6)
    tha = (0.02 * rng.standard_normal(N)).astype(np.float32)
    thb = tha.copy()
    for g in make_grads(rng, N, R, 4):
        a.step(tha, g)
        b.step(thb, g)
        assert b.last_coef() == 1.0
        assert np.array_equal(tha.view(np.uint32), thb.view(np.uint32))
        np.testing.assert_allclose(b.last_norm(), np.sqrt(np.sum(b.ghat().astype(np.float64) ** 2)), rtol=1e-12)


def test_p11_clip_scales_only_the_second_moment_input_sparse():
    """On a sparse step: m_t = b-bar is unchanged by the clip (l.12 precedes l.14); g-hat is scaled by
    coef = c / (||g-hat|| + 1e-6); off-mask parameters are untouched by it."""
    rng = np.random.default_rng(15)
    N, R = 3000, 2
    a, b = ScapeOracle(N, R, 0.9, **HYP), ScapeOracle(N, R, 0.9, **HYP)
    b.set_clip_grad(1e-3)
    tha = (0.02 * rng.standard_normal(N)).astype(np.float32)
    thb = tha.copy()
    gs = make_grads(rng, N, R, 3)
    for g in gs[:2]:
        a.step(tha, g)
        b.set_clip_grad(0.0); b.step(thb, g); b.set_clip_grad(1e-3)      # identical history
    a.step(tha, gs[2]); b.step(thb, gs[2])
    assert b.last_coef() < 1.0
    np.testing.assert_array_equal(a.m(), b.m())
    np.testing.assert_allclose(b.ghat(), a.ghat() * np.float32(b.last_coef()), rtol=2e-7)
    np.testing.assert_allclose(b.last_coef(), 1e-3 / (a.last_norm() + 1e-6), rtol=1e-6)
    off = np.ones(N, bool); off[a.idx()] = False
    np.testing.assert_array_equal(tha[off], thb[off])
    assert not np.array_equal(tha[~off], thb[~off])


# ------------------------------------------------------------------------------------ P12
def layered_brute_force(x, offsets, compress, s):
    """Per-layer refresh written from the definition: inside each compressed layer the
    k_l = n_l - floor(s n_l) entries of largest |x| (ties to the lower index), every entry of an
    uncompressed layer."""
    mask = np.zeros(len(x), np.uint8)
    for l in range(len(offsets) - 1):
        a, b = offsets[l], offsets[l + 1]
        if not compress[l]:
            mask[a:b] = 1
        else:
            n = b - a
            mask[a:b] = brute_force_topk(x[a:b], n - int(np.floor(s * n)))
    return mask


@pytest.mark.parametrize("seed", range(4))
def test_p12_per_layer_refresh_vs_brute_force(seed):
    rng = np.random.default_rng(100 + seed)
    N, R = 300, 2
    cuts = np.sort(rng.choice(np.arange(1, N), size=5, replace=False))
    offsets = np.concatenate([[0], cuts, [N]])
    compress = np.array([1, 1, 0, 1, 1, 1], np.uint8)
    s = [0.9, 0.5, 0.75, 0.99][seed]
    o = ScapeOracle(N, R, s, **HYP)
    o.set_layers(offsets, compress)
    th = (0.02 * rng.standard_normal(N)).astype(np.float32)
    scale = np.repeat(10.0 ** rng.uniform(-3, 0, 6), np.diff(offsets)).astype(np.float32)
    for g in make_grads(rng, N, R, 4):
        g = [x * scale for x in g]
        if seed == 0:                      # ties inside and across layers
            g = [np.round(x * 2e3) / 2e3 for x in g]
        o.step(th, g)
        mk = o.mask()
        np.testing.assert_array_equal(mk, layered_brute_force(o.mt(0), offsets, compress, s))
        for l in range(6):                 # exactly k_l per layer
            n = offsets[l + 1] - offsets[l]
            want = n if not compress[l] else n - int(np.floor(s * n))
            assert mk[offsets[l]:offsets[l + 1]].sum() == want


def test_p12_one_layer_is_the_flat_refresh_and_layers_differ_from_flat():
    rng = np.random.default_rng(12)
    N, R, T = 2000, 2, 5
    grads = make_grads(rng, N, R, T)
    th0 = (0.02 * rng.standard_normal(N)).astype(np.float32)
    flat = ScapeOracle(N, R, 0.9, **HYP)
    one = ScapeOracle(N, R, 0.9, **HYP)
    one.set_layers([0, N])
    two = ScapeOracle(N, R, 0.9, **HYP)
    two.set_layers([0, 700, N])
    tha, thb, thc = th0.copy(), th0.copy(), th0.copy()
    scale = np.where(np.arange(N) < 700, 1.0, 30.0).astype(np.float32)   # a flat top-k would starve layer 0
    for g in grads:
        g = [x * scale for x in g]
        flat.step(tha, g); one.step(thb, g); two.step(thc, g)
        np.testing.assert_array_equal(flat.mask(), one.mask())
        assert np.array_equal(tha.view(np.uint32), thb.view(np.uint32))
        assert two.mask()[:700].sum() == 70 and two.mask()[700:].sum() == 130
    assert flat.mask()[:700].sum() < 70


def test_set_layers_rejects_bad_offsets():
    o = ScapeOracle(100, 1, 0.5, **HYP)
    for bad in ([0, 50], [1, 100], [0, 50, 50, 100], [0, 60, 40, 100]):
        with pytest.raises(ValueError):
            o.set_layers(bad)
    with pytest.raises(ValueError):
        o.set_sparsity(1.0)


# ------------------------------------------------------------------------------------ P13
def test_p13_uncompressed_layer_is_dense_adams_on_its_slice_double():
    """A layer that is not sparsified stays in every mask, so on its slice
    e = 0 and the step is Eq. 2 with the replica-mean gradient."""
    rng = np.random.default_rng(13)
    N, R, T = 1200, 3, 7
    a, b = 500, 640
    o = ScapeOracle(N, R, 0.95, dtype=np.float64, **HYP)
    o.set_layers([0, a, b, N], [1, 0, 1])
    th = 0.02 * rng.standard_normal(N)
    th_ref, m_ref = th[a:b].copy(), np.zeros(b - a)
    for g in make_grads(rng, N, R, T, dtype=np.float64):
        o.step(th, g)
        gbar = sum(x[a:b] for x in g) / R
        th_ref, m_ref = dense_adams_f64(th_ref, m_ref, gbar, **HYP)
        assert o.mask()[a:b].all()
        for r in range(R):
            assert not o.e(r)[a:b].any()
        np.testing.assert_allclose(o.m()[a:b], m_ref, rtol=1e-12, atol=1e-300)
        np.testing.assert_allclose(th[a:b], th_ref, rtol=1e-12, atol=1e-300)
    # the sparsified layers hold exactly their k_l
    assert o.mask()[:a].sum() == a - int(np.floor(0.95 * a))
    assert o.mask()[b:].sum() == (N - b) - int(np.floor(0.95 * (N - b)))


# ------------------------------------------------------------------------------------ P14
def warmup_density(t, d_final, T_w):
    """Exponential density warm-up 1 -> d_final over T_w steps (PAPER.md:279 gives the shape only)."""
    return max(d_final, d_final ** (t / T_w))


def test_p14_sparsity_schedule_counts_delay_and_conservation_double():
    rng = np.random.default_rng(14)
    N, R, T = 1000, 2, 12
    offsets, compress = [0, 300, 364, N], [1, 0, 1]
    o = ScapeOracle(N, R, 0.0, dtype=np.float64, **HYP)
    o.set_layers(offsets, compress)
    th = 0.02 * rng.standard_normal(N)
    c1 = 1 - HYP["beta1"]
    sum_g, sum_m_before = np.zeros(N), np.zeros(N)
    want_prev = N                                   # M_0 = 1
    for t, g in enumerate(make_grads(rng, N, R, T, dtype=np.float64), start=1):
        s = 1.0 - warmup_density(t, 0.05, 8)
        o.set_sparsity(s)                           # used by this step's refresh (M_t)
        sum_m_before += o.m()
        o.step(th, g)
        assert o.K_last == want_prev                # the step used the mask made one step earlier
        want_prev = sum((b - a) if not c else (b - a) - int(np.floor(s * (b - a)))
                        for a, b, c in zip(offsets[:-1], offsets[1:], compress))
        assert o.mask().sum() == want_prev
        np.testing.assert_array_equal(o.mask(), layered_brute_force(o.mt(0), offsets, compress, s))
        # P6 under a changing mask size: nothing is lost
        sum_g += sum(g) / R
        ebar = sum(o.e(r) for r in range(R)) / R
        np.testing.assert_allclose(c1 * sum_g, ebar + o.m() + c1 * sum_m_before, rtol=1e-10, atol=1e-14)
    assert want_prev == 15 + 64 + 32               # 5 % of 300 and of 636, all 64 of the uncompressed layer


# ---------------------------------------------------------------------------------------------
# P15 workers ("N workers"; §IV-A :178 "each worker only computes a portion of the
# top-k operations ... the new local masks from all workers are gathered")
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("W,Rl", [(2, 1), (2, 2), (4, 1), (3, 2)])
def test_p15_every_layer_follows_its_owner_and_the_two_level_mean(W, Rl):
    rng = np.random.default_rng(1500 + 10 * W + Rl)
    N, R, s = 400, W * Rl, 0.9
    cuts = np.sort(rng.choice(np.arange(1, N), size=5, replace=False))
    offsets = np.concatenate([[0], cuts, [N]])
    compress = np.array([1, 1, 1, 0, 1, 1], np.uint8)
    owner = np.array([l % W for l in range(6)], np.int32)
    o = ScapeOracle(N, R, s, **HYP, dtype=np.float64)
    o.set_layers(offsets, compress)
    o.set_workers(W, owner)
    th = 0.02 * rng.standard_normal(N)
    for g in make_grads(rng, N, R, 5, dtype=np.float64):
        # replicas that disagree strongly, so that the owner matters
        g = [x * (1.0 + 3.0 * r) for r, x in enumerate(g)]
        o.step(th, g)
        mk = o.mask()
        want = np.zeros(N, np.uint8)
        for l in range(6):                       # brute force inside the layer on ITS OWNER's statistic
            a, b = offsets[l], offsets[l + 1]
            if not compress[l]:
                want[a:b] = 1
                continue
            x = o.mt(int(owner[l]) * Rl)[a:b]
            want[a:b] = brute_force_topk(x, (b - a) - int(np.floor(s * (b - a))))
        np.testing.assert_array_equal(mk, want)
        # l.10: the two-level sum is the mean over all R replicas
        flat = np.mean(np.stack([o.b(r) for r in range(R)]), axis=0)
        np.testing.assert_allclose(o.bbar(), flat, rtol=1e-12, atol=1e-18)   # sums may cancel
    # a different owner gives a different mask (the pin has teeth)
    assert not np.array_equal(want, layered_brute_force(o.mt(0), offsets, compress, s))


def test_p15_one_worker_or_one_replica_per_worker_is_the_plain_step_fp32():
    rng = np.random.default_rng(1515)
    N, R, T = 500, 4, 5
    offsets = [0, 100, 333, N]
    grads = make_grads(rng, N, R, T)
    th0 = (0.02 * rng.standard_normal(N)).astype(np.float32)
    plain = ScapeOracle(N, R, 0.9, **HYP); plain.set_layers(offsets)
    one = ScapeOracle(N, R, 0.9, **HYP); one.set_layers(offsets); one.set_workers(1)
    # R workers of one replica each, all layers owned by worker 0: the same left-to-right sum
    per = ScapeOracle(N, R, 0.9, **HYP); per.set_layers(offsets); per.set_workers(R, [0, 0, 0])
    tha, thb, thc = th0.copy(), th0.copy(), th0.copy()
    for g in grads:
        plain.step(tha, g); one.step(thb, g); per.step(thc, g)
        for o in (one, per):
            np.testing.assert_array_equal(o.mask(), plain.mask())
            assert np.array_equal(o.bbar().view(np.uint32), plain.bbar().view(np.uint32))
    assert np.array_equal(tha.view(np.uint32), thb.view(np.uint32))
    assert np.array_equal(tha.view(np.uint32), thc.view(np.uint32))


def test_p15_set_workers_rejects_bad_arguments():
    o = ScapeOracle(64, 4, 0.5, **HYP)
    with pytest.raises(ValueError):
        o.set_workers(3)                         # R not divisible
    with pytest.raises(ValueError):
        o.set_workers(2, [0, 1])                 # owners need layers
    o.set_layers([0, 32, 64])
    with pytest.raises(ValueError):
        o.set_workers(2, [0, 2])                 # owner out of range
    o.set_workers(2, [1, 0])


# ---------------------------------------------------------------------------------------------
# P16 mask bit pack / unpack: the oracle's plain loop against numpy's packbits
# (a library routine, another route to the same definition), a hand-written example, the round trip
# ---------------------------------------------------------------------------------------------
def test_p16_mask_pack_unpack():
    from oracle.scape_oracle import mask_pack, mask_unpack
    # by hand: entries 0, 5, 31 -> word 0 = 1 + 32 + 2^31; entry 32 -> word 1 bit 0; entry 70 -> word 2 bit 6
    m = np.zeros(71, np.uint8); m[[0, 5, 31, 32, 70]] = [1, 9, 255, 1, 1]
    np.testing.assert_array_equal(mask_pack(m), np.array([1 + 32 + 2**31, 1, 64], np.uint32))
    rng = np.random.default_rng(16)
    for n in (1, 31, 32, 33, 64, 1000, 4099):
        m = (rng.random(n) < 0.3).astype(np.uint8) * rng.integers(1, 255, n).astype(np.uint8)
        w = mask_pack(m)
        lib = np.packbits(np.concatenate([m != 0, np.zeros((-n) % 32, bool)]), bitorder="little").view(np.uint32)
        np.testing.assert_array_equal(w, lib)
        np.testing.assert_array_equal(mask_unpack(w, n), (m != 0).astype(np.uint8))
        assert w.size == (n + 31) // 32


# ------------------------------------------------------------------------------------ P17-P20
# Algorithm 2, parameter side (PAPER.md:222-242; Eq. 6 :207-211; "Use FP32 w", :231-232)
def test_p17_bf16_round_to_nearest_even_vs_torch_and_crafted_ties():
    """The oracle's float -> bfloat16 (written out from the definition) against (i) the torch CPU
    conversion, a library routine, on random values of every magnitude, denormals, +-0, +-inf, and
    (ii) hand-checked ties: exactly half goes to the even neighbour, anything above half goes up."""
    import torch
    from oracle.scape_oracle import bf16_rne, bf16_widen
    rng = np.random.default_rng(17)
    bits = rng.integers(0, 2**32, 400_000, dtype=np.uint64).astype(np.uint32)
    x = bits.view(np.float32)
    x = x[np.isfinite(x)]
    x = np.concatenate([x, np.array([0.0, -0.0, np.inf, -np.inf, 1e-45, -1e-45, 1e-40, 3.3895314e38, -3.4e38], np.float32),
                        (1e-3 * rng.standard_normal(100_000)).astype(np.float32)])
    got = bf16_rne(x)
    want = torch.from_numpy(x.copy()).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    np.testing.assert_array_equal(got, want)
    # (ii) by hand: bf16 keeps 8 significant bits
    cases = {1.0: 1.0, 1.0 + 2.0**-8: 1.0, 1.0 + 2.0**-8 + 2.0**-23: 1.0 + 2.0**-7, 1.0 + 2.0**-7 + 2.0**-8: 1.0 + 2.0**-6,
             1.0 + 2.0**-7: 1.0 + 2.0**-7, -(1.0 + 2.0**-8 + 2.0**-16): -(1.0 + 2.0**-7), 2.0 - 2.0**-9: 2.0,
             2.0 - 2.0**-8: 2.0, 2.0 - 2.0**-8 - 2.0**-20: 2.0 - 2.0**-7}
    xs = np.array(list(cases), np.float32)
    np.testing.assert_array_equal(bf16_widen(bf16_rne(xs)), np.array(list(cases.values()), np.float32))
    # widening is exact and rounding a bf16 value is the identity
    b = rng.integers(0, 2**16, 5000).astype(np.uint16)
    b = b[np.isfinite(bf16_widen(b))]
    np.testing.assert_array_equal(bf16_rne(bf16_widen(b)), b)


def test_p19_alg2_parameter_hand_example():
    """tests/golden/p19_alg2_param_example.json: 8 parameters, dyadic values, worked by hand."""
    from oracle.scape_oracle import bf16_rne, bf16_widen, param_apply, param_pack
    with open(os.path.join(HERE, "golden", "p19_alg2_param_example.json")) as f:
        G = json.load(f)
    mask = np.array(G["mask"], np.uint8)
    th = np.array(G["theta_owner"], np.float32)
    pf = param_pack(th, mask, "f32")
    pb = param_pack(th, mask, "bf16")
    np.testing.assert_array_equal(pf, np.array(G["pack_f32"], np.float32))          # ascending index order
    np.testing.assert_array_equal(bf16_widen(pb), np.array(G["pack_bf16_as_f32"], np.float32))
    for payload, tag in ((pf, "f32"), (pb, "bf16")):
        for form in (0, 1):                              # l.17 with u = 0 and Eq. 6 literally: identical here (all exact)
            w = np.array(G["w_before"], np.float32)
            w_hat = np.zeros(G["N"], np.uint16)
            param_apply(w, mask, payload, G["lr"], G["wd"], w_hat=w_hat, form=form)
            np.testing.assert_array_equal(w, np.array(G[f"w_after_{tag}_payload"], np.float32))
            np.testing.assert_array_equal(bf16_widen(w_hat), np.array(G[f"w_hat_after_{tag}_payload_as_f32"], np.float32))


def test_p20_eq6_literal_vs_l17_with_u_zero_within_one_ulp():
    """Eq. 6: theta[not M] = (1 - eta lambda) theta.  The graded form is Alg. 1 l.17
    with u = 0, fma(-eta, lambda*theta, theta) (readings S13, S21); the two differ by at most 1 ulp, and
    both agree with the exact product to 1 ulp."""
    from oracle.scape_oracle import param_apply
    rng = np.random.default_rng(20)
    N = 200_000
    w0 = (0.02 * rng.standard_normal(N)).astype(np.float32)
    w0[:7] = [0.0, -0.0, 1e-40, -1e-38, 3e38, 1.0, -1.0]
    mask = np.zeros(N, np.uint8)
    for lr, wd in ((1e-3, 0.1), (3e-4, 0.1), (1.5e-4, 0.01), (0.5, 0.25)):
        a, b = w0.copy(), w0.copy()
        param_apply(a, mask, np.zeros(0, np.float32), lr, wd, form=0)
        param_apply(b, mask, np.zeros(0, np.float32), lr, wd, form=1)
        exact = (1.0 - np.float64(np.float32(lr)) * np.float64(np.float32(wd))) * w0.astype(np.float64)
        assert np.all(np.abs(a.astype(np.float64) - b.astype(np.float64)) <= ulp32(exact))
        assert np.all(np.abs(a.astype(np.float64) - exact) <= ulp32(exact))
        assert np.all(np.abs(b.astype(np.float64) - exact) <= ulp32(exact))
        assert np.array_equal(np.signbit(a), np.signbit(w0))


@pytest.mark.parametrize("R,sparsity", [(2, 0.9), (1, 0.99), (3, 0.0)])
def test_p18_alg2_copy_tracks_the_owner_bitwise(R, sparsity):
    """Algorithm 2 l.2-4 with Algorithm 1 as the owner's update.  The owner steps theta with the SCAPE
    step; a non-owner keeps the FP32 copy w and the bf16 compute copy w^ and, after every step, gets the
    owner's theta on the mask THAT STEP USED (M_{t-1}: Eq. 6, reading S22) and decays the rest locally.
      fp32 payload: w == theta bit for bit after every step, w^ == bf16(theta) everywhere;
      bf16 payload: w^ == bf16(theta) on the mask, w == widen(bf16(theta)) there;
      wrong mask (the refreshed M_t instead of M_{t-1}): the copy drifts at once -- the pin has teeth."""
    from oracle.scape_oracle import bf16_rne, bf16_widen, param_apply, param_pack
    rng = np.random.default_rng(18 + R)
    N, T = 3001, 6
    grads = make_grads(rng, N, R, T)
    ora = ScapeOracle(N, R, sparsity, **HYP)
    theta = (0.02 * rng.standard_normal(N)).astype(np.float32)
    w = theta.copy()                       # the non-owner starts from the same parameters
    w_bf = theta.copy()                    # a second copy fed with bf16 payloads
    w_wrong = theta.copy()
    drifted = False
    for t in range(T):
        used = ora.mask().copy()           # M_{t-1}: the mask the coming step uses
        ora.step(theta, grads[t])
        refreshed = ora.mask()             # M_t
        # fp32 payload
        w_hat = np.zeros(N, np.uint16)
        param_apply(w, used, param_pack(theta, used, "f32"), HYP["lr"], HYP["wd"], w_hat=w_hat)
        assert np.array_equal(w.view(np.uint32), theta.view(np.uint32)), f"step {t + 1}: the FP32 copy left the owner's theta"
        np.testing.assert_array_equal(w_hat, bf16_rne(theta))
        # bf16 payload
        w_hat_b = np.zeros(N, np.uint16)
        pb = param_pack(theta, used, "bf16")
        np.testing.assert_array_equal(pb, bf16_rne(theta[used.astype(bool)]))
        param_apply(w_bf, used, pb, HYP["lr"], HYP["wd"], w_hat=w_hat_b)
        on = used.astype(bool)
        np.testing.assert_array_equal(w_hat_b[on], bf16_rne(theta[on]))
        np.testing.assert_array_equal(w_bf[on], bf16_widen(bf16_rne(theta[on])))
        # the wrong mask
        if sparsity > 0 and t >= 1:
            param_apply(w_wrong, refreshed, param_pack(theta, refreshed, "f32"), HYP["lr"], HYP["wd"])
            drifted = drifted or not np.array_equal(w_wrong, theta)
        else:
            w_wrong[:] = theta
    if sparsity > 0:
        assert drifted, "exchanging on M_t instead of M_{t-1} went unnoticed"
