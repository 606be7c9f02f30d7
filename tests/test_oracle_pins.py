"""Pins for the CPU oracle (oracle/lpf_oracle.cpp): each test checks an oracle
function against something OTHER than itself -- a closed form, a SciPy/NumPy
routine it must reduce to, an invariant, a hand example, brute force on a tiny
input, or an injected source of known position and flux ("What
pins each part").  A dropped term, wrong sign or index, or transposed operand in
the oracle fails at least one of these.
"""
import math
import os

import numpy as np
import pytest
import scipy.ndimage as ndi
import scipy.stats as sst

import oracle as O
from paper_2103_15418_b200 import synth

GOLD = os.path.join(os.path.dirname(__file__), "golden")
SIG = synth.SIGMA_SRC


def P(**kw):
    p = dict(kappa=5.0, k_max=2, eps_rel=1e-5, sigma_mf=0.85, k_mf=3, bg_kernel=1, s_bg=8.0, k_bg=12,
             n_iter=1, detect_sum_plane=1, qc_tau=5.0, qc_clip=3.0, r_flux=1, r_dedupe=2, r_assoc=3,
             n_forget=10, T_ring=8, n_cand_max=32, max_det=1024)
    p.update(kw)
    return p


def gauss_img(D, y0, x0, A, sig):
    yy, xx = np.mgrid[:D, :D]
    return A * np.exp(-((yy - y0) ** 2 + (xx - x0) ** 2) / (2 * sig ** 2))


# ---------------------------------------------------------------- O1 / O2 ----
def test_band_stats_reduce_to_numpy():
    rng = np.random.default_rng(0)
    cube = (rng.standard_normal((3, 40, 50)) * [[[1.0]], [[2.5]], [[0.3]]] + [[[0.0]], [[7.0]], [[-2.0]]]).astype(np.float32)
    W = (rng.random((40, 50)) > 0.3).astype(np.uint8)
    st = O.band_stats(cube, W, 3.0)
    for b in range(3):
        v = cube[b][W == 1].astype(np.float64)
        assert st[b, 0] == v.size
        assert abs(st[b, 1] - v.mean()) < 1e-12
        assert abs(st[b, 2] - v.std()) < 1e-12
        keep = v[np.abs(v - v.mean()) <= 3.0 * v.std()]      # O1: the plain float64 definition
        assert st[b, 3] == keep.size and keep.size < v.size
        assert abs(st[b, 4] - keep.mean()) < 1e-12 and abs(st[b, 5] - keep.std()) < 1e-12
    # no mask == all-ones mask
    assert np.allclose(O.band_stats(cube, None, 3.0), O.band_stats(cube, np.ones((40, 50), np.uint8), 3.0))


def _stats_from(means, rms, n=1e6):
    st = np.zeros((len(means), 6))
    st[:, 0] = n; st[:, 1] = means; st[:, 2] = rms
    return st


def test_verdict_hand_example():
    # eq. A.1 on b = (1,2,3,4,100): median 3, MAD 1 -> z = (-2,-1,0,1,97)
    z, ok = O.qc_verdict(_stats_from([1, 2, 3, 4, 100], [1e-3] * 5), 5.0)
    assert np.allclose(z[:, 0], [-2, -1, 0, 1, 97], atol=1e-12)
    assert np.allclose(z[:, 1], 0)
    assert ok.tolist() == [1, 1, 1, 1, 0, 1]


def test_verdict_matches_scipy_mad_and_invariances():
    rng = np.random.default_rng(3)
    for B in (4, 5, 16, 64):
        v = rng.standard_normal(B) * 3 + 10
        r = np.abs(rng.standard_normal(B)) + 5
        z, ok = O.qc_verdict(_stats_from(v, r * 1e-6, n=1e12), 5.0)   # SE floor negligible
        mad = sst.median_abs_deviation(v, scale=1.0)
        assert np.allclose(z[:, 0], (v - np.median(v)) / mad, rtol=1e-12)
        mad_r = sst.median_abs_deviation(r, scale=1.0)
        assert np.allclose(z[:, 1], (r - np.median(r)) / mad_r, rtol=1e-9)
        # affine invariance of z (a > 0) and permutation equivariance
        z2, _ = O.qc_verdict(_stats_from(2.5 * v - 4.0, r * 1e-6, n=1e12), 5.0)
        assert np.allclose(z2[:, 0], z[:, 0], rtol=1e-9)
        perm = rng.permutation(B)
        z3, ok3 = O.qc_verdict(_stats_from(v[perm], (r * 1e-6)[perm], n=1e12), 5.0)
        assert np.allclose(z3, z[perm], rtol=1e-12) and np.array_equal(ok3[:-1], ok[perm])


def test_verdict_se_floor_and_degenerate():
    # identical bands: MAD = 0 -> floor at SE = median(rms)/sqrt(n)  (reading R12)
    z, ok = O.qc_verdict(_stats_from([0.0, 0.0, 0.0, 0.004], [1.0] * 4, n=1e6), 5.0)
    assert abs(z[3, 0] - 0.004 / (1.0 / 1e3)) < 1e-9 and ok.tolist() == [1, 1, 1, 1, 1]
    z, ok = O.qc_verdict(_stats_from([0.0, 0.0, 0.0, 0.006], [1.0] * 4, n=1e6), 5.0)
    assert ok.tolist() == [1, 1, 1, 0, 1]
    # rms vector: SE_rms = median(rms)/sqrt(2n)
    z, ok = O.qc_verdict(_stats_from([0.0] * 4, [1.0, 1.0, 1.0, 1.0 + 0.01], n=1e6), 5.0)
    assert abs(z[3, 1] - 0.01 / (1.0 / math.sqrt(2e6))) < 1e-6 and ok[3] == 0
    # constant cube: everything 0/0 -> z = 0, all ok
    z, ok = O.qc_verdict(_stats_from([2.0] * 4, [0.0] * 4), 5.0)
    assert np.all(z == 0) and ok.tolist() == [1, 1, 1, 1, 1]
    # non-finite band is rejected and ignored by the medians; majority rule for frame_ok
    st = _stats_from([1, 2, 3, 4, np.nan], [1e-3] * 5)
    z, ok = O.qc_verdict(st, 5.0)
    assert ok.tolist() == [1, 1, 1, 1, 0, 1]
    z, ok = O.qc_verdict(_stats_from([0, 0, 50, 90, -70, 30], [1e-3] * 6), 5.0)
    assert ok[-1] == (ok[:-1].sum() >= 3)


def test_qc_flags_injected_rfi_and_keeps_clean_bands():
    # both corruption modes of config 3 on a reduced-size frame
    rng = np.random.default_rng(5)
    D, B = 256, 16
    W = synth.horizon_mask(D)
    sig = (synth.noise_sigma_map(D) * W).astype(np.float32)
    for trial in range(4):
        cube = rng.standard_normal((B, D, D), dtype=np.float32) * sig
        cube[3] *= 10.0
        rows = rng.integers(30, 220, size=2)
        cube[9, rows, :] += 20.0 * sig[rows, :]
        st = O.band_stats(cube, W, 3.0)
        z, ok = O.qc_verdict(st, 5.0)
        assert ok[3] == 0 and ok[9] == 0
        assert ok[[b for b in range(B) if b not in (3, 9)]].all() and ok[B] == 1


# ---------------------------------------------------------------- O3 ---------
def test_gauss_taps_golden_and_normalised():
    for line in open(os.path.join(GOLD, "gauss_taps.txt")):
        if line.startswith("#") or not line.strip():
            continue
        tok = line.split()
        s, k, vals = float(tok[0]), int(tok[1]), [float(v) for v in tok[2:]]
        g = O.kernel_taps(0, s, k)
        assert g.size == 2 * k + 1 and abs(g.sum() - 1) < 1e-15
        assert np.allclose(g, g[::-1], atol=0)
        assert np.allclose(g[:k + 1], vals, atol=5e-10)
    assert np.allclose(O.kernel_taps(1, 0.0, 12), 1 / 25.0)
    assert O.kernel_taps(0, 0.0, 3).tolist() == [0, 0, 0, 1, 0, 0, 0]


@pytest.mark.parametrize("direct", [True, False])
def test_delta_image_gives_kernel(direct):
    # a delta image convolved equals the kernel (north_star pin), to 1 ulp-level in float64
    for (kind, s, k) in [(0, 0.85, 3), (0, 8.0, 16), (1, 0.0, 12)]:
        g = O.kernel_taps(kind, s, k)
        D = 4 * k + 5   # every output inside the delta's footprint has its full window in the image
        A = np.zeros((D, D)); A[D // 2, D // 2 + 1] = 1.0
        out = O.normconv(A, None, g, direct=direct)
        G = np.outer(g, g)
        y0, x0 = D // 2, D // 2 + 1
        win = out[y0 - k:y0 + k + 1, x0 - k:x0 + k + 1]
        assert np.allclose(win, G[::-1, ::-1], rtol=2e-13, atol=0)   # (the sum of the weights is 1 to rounding)
        assert abs(out.sum() - 1) < 1e-12
        outside = out.copy(); outside[y0 - k:y0 + k + 1, x0 - k:x0 + k + 1] = 0
        assert np.all(outside == 0)


def test_normconv_reduces_to_scipy_in_the_interior():
    rng = np.random.default_rng(1)
    A = rng.standard_normal((70, 83))
    for (s, k) in [(0.85, 3), (8.0, 16)]:
        g = O.kernel_taps(0, s, k)
        ref = ndi.gaussian_filter(A, sigma=s, truncate=k / s, mode="constant")
        out = O.normconv(A, None, g, direct=True)
        assert np.allclose(out[k:-k, k:-k], ref[k:-k, k:-k], rtol=1e-12, atol=1e-13)
        # at the border scipy zero-pads; the oracle renormalises (reading R7): ratio = denominator
        out2, den = O.normconv(A, None, g, direct=True, want_den=True)
        assert np.allclose(out2 * den, ref, rtol=1e-11, atol=1e-12)
    K = 12
    ref = ndi.uniform_filter(A, size=2 * K + 1, mode="constant")
    out, den = O.normconv(A, None, O.kernel_taps(1, 0, K), want_den=True)
    assert np.allclose(out * den, ref, rtol=1e-11, atol=1e-12)
    assert np.allclose(den[K:-K, K:-K], 1.0)


def test_normconv_asymmetric_kernel_orientation_and_axes():
    # a transposed operand or swapped axis in the oracle fails here
    A = np.zeros((9, 11)); A[4, 5] = 1.0; A[2, 8] = 2.0
    g = np.array([0.1, 0.2, 0.7])  # asymmetric taps: correlation form out(n,m) = sum g_j g_i A(n+j, m+i)
    out = O.normconv(A, None, g, direct=True)
    ref = ndi.correlate1d(ndi.correlate1d(A, g, axis=1, mode="constant"), g, axis=0, mode="constant")
    den = ndi.correlate1d(ndi.correlate1d(np.ones_like(A), g, axis=1, mode="constant"), g, axis=0, mode="constant")
    assert np.allclose(out, ref / den, rtol=1e-13)
    assert np.allclose(O.normconv(A, None, g, direct=False), out, rtol=1e-13)


def test_normconv_direct_equals_factorised_with_masks():
    rng = np.random.default_rng(2)
    A = rng.standard_normal((61, 57)) + 3.0
    W = (rng.random((61, 57)) > 0.4).astype(np.uint8)
    W[10:30, 10:40] = 0  # a hole larger than the small kernel
    for (kind, s, k) in [(0, 0.85, 3), (0, 8.0, 16), (1, 0.0, 12)]:
        g = O.kernel_taps(kind, s, k)
        a, da = O.normconv(A, W, g, direct=True, want_den=True)
        b, db = O.normconv(A, W, g, direct=False, want_den=True)
        assert np.allclose(a, b, rtol=1e-11, atol=1e-13) and np.allclose(da, db, rtol=1e-12, atol=1e-15)
        # definition: weighted mean over valid pixels -> constants are reproduced wherever den > 0
        c = O.normconv(np.full_like(A, 4.25), W, g, direct=True)
        assert np.allclose(c[da > 0], 4.25, rtol=1e-13) and np.all(c[da == 0] == 0)
    # brute force of the definition at a few pixels
    g = O.kernel_taps(0, 2.0, 4)
    a = O.normconv(A, W, g, direct=True)
    for (y, x) in [(0, 0), (5, 56), (33, 20), (60, 3)]:
        num = den = 0.0
        for j in range(-4, 5):
            for i in range(-4, 5):
                yy, xx = y + j, x + i
                if 0 <= yy < 61 and 0 <= xx < 57 and W[yy, xx]:
                    num += g[j + 4] * g[i + 4] * A[yy, xx]; den += g[j + 4] * g[i + 4]
        assert abs(a[y, x] - (num / den if den > 0 else 0.0)) < 1e-13


# ---------------------------------------------------------------- O4 ---------
def test_planes_and_sum_plane():
    rng = np.random.default_rng(4)
    cube = rng.standard_normal((4, 6, 7)).astype(np.float32)
    ok = np.array([1, 0, 1, 1, 1], np.uint8)
    pl = O.planes(cube, ok)
    assert np.array_equal(pl[0], cube[0].astype(np.float64)) and np.all(pl[1] == 0)
    assert np.allclose(pl[4], cube[0].astype(np.float64) + cube[2] + cube[3], atol=1e-15)


def test_matched_filter_noise_gain_and_source_gain():
    p = P()
    rng = np.random.default_rng(6)
    X = rng.standard_normal((200, 200))
    d = O.detect_plane(X, None, p, direct=False)
    g = O.kernel_taps(0, 0.85, 3)
    assert abs((g ** 2).sum() - 0.33242) < 1e-5                 # closed form
    assert abs(d["F"][10:-10, 10:-10].std() - (g ** 2).sum()) < 0.01
    # FWHM-2 source of amplitude A: peak after g_mf = A (sum_i g_i exp(-i^2/2 sig^2))^2  (~0.5012 A)
    A = 7.0
    Fs = O.detect_plane(gauss_img(41, 20, 20, A, SIG), None, p)["F"]
    i = np.arange(-3, 4)
    gain = (g * np.exp(-i ** 2 / (2 * SIG ** 2))).sum() ** 2
    assert abs(gain - 0.5012) < 2e-4 and abs(Fs[20, 20] - A * gain) < 1e-12
    assert abs(gain - SIG ** 2 / (SIG ** 2 + 0.85 ** 2)) < 5e-3  # continuum closed form 0.4996


# ---------------------------------------------------------------- O5 ---------
def test_constant_and_affine_images():
    for bg in (dict(bg_kernel=1, k_bg=12), dict(bg_kernel=0, s_bg=8.0, k_bg=16)):
        for n_iter in (1, 3):
            p = P(n_iter=n_iter, **bg)
            rng = np.random.default_rng(7)
            W = (rng.random((60, 64)) > 0.2).astype(np.uint8)
            for c in (0.0, 1.0, 0.1, -3.7, 1e6, 1e-20):
                for mask in (None, W):
                    d = O.detect_plane(np.full((60, 64), c), mask, p)
                    assert d["P"].sum() == 0 and d["iter"].sum() == 0       # constant image -> zero detections
                    v = d["C_last"][mask == 1] if mask is not None else d["C_last"]
                    assert np.allclose(v, c, rtol=1e-12, atol=0)
                    assert np.all(np.abs(d["S_last"]) <= (1e-12 * abs(c)) ** 2 + 1e-300)
    # affine image: C = X and S = 0 in the interior (symmetric kernel), no detections anywhere
    yy, xx = np.mgrid[:90, :90]
    X = 0.3 * xx + 0.7 * yy + 5.0
    pp = P(sigma_mf=0.0)
    d = O.detect_plane(X, None, pp)
    k = 12
    assert np.allclose(d["C_last"][k:-k, k:-k], X[k:-k, k:-k], rtol=1e-13)
    k2 = 2 * k
    assert np.all(d["S_last"][k2:-k2, k2:-k2] < 1e-20)
    assert d["P"][k2:-k2, k2:-k2].sum() == 0


def test_gaussian_source_closed_forms_gauss_bg():
    # noiseless Gaussian source (sigma, A) under Gaussian G (s, k >= 4 s), sigma_mf = 0:
    # C0 = A a/(a+b);  S0 = A^2 [ (a/2)/(a/2+b) + (a/(a+b))^2 v2/(v2+b) - 2 (a/(a+b)) v3/(v3+b) ]
    sig, s, A = 1.2015, 4.0, 9.0
    k = 16
    D = 101
    X = gauss_img(D, 50, 50, A, sig)
    d = O.detect_plane(X, None, P(sigma_mf=0.0, bg_kernel=0, s_bg=s, k_bg=k), direct=False)
    a, b = sig ** 2, s ** 2
    C0 = A * a / (a + b)
    v2, v3 = (a + b) / 2, a * (a + b) / (2 * a + b)
    S0 = A ** 2 * ((a / 2) / (a / 2 + b) + (a / (a + b)) ** 2 * v2 / (v2 + b) - 2 * (a / (a + b)) * v3 / (v3 + b))
    assert abs(d["C_last"][50, 50] - C0) / C0 < 2e-4
    assert abs(d["S_last"][50, 50] - S0) / S0 < 2e-4
    # bright-limit margin (x-c)/sqrt(S) ~ s sqrt2 / sigma_src (SURVEY reading 3), kernel-truncation tolerant
    m = (A - d["C_last"][50, 50]) / math.sqrt(d["S_last"][50, 50])
    assert abs(m - (A - C0) / math.sqrt(S0)) / m < 2e-4


def test_gaussian_source_closed_forms_box_bg():
    # BOX K: C0 = 2 pi sigma^2 A / (2K+1)^2 ; bright-limit margin ~ (2K+1)/(sigma sqrt(pi))
    K, A = 12, 11.0
    for sig, margin in ((SIG, 16.6), (1.2015, 11.8)):
        X = gauss_img(81, 40, 40, A, sig)
        d = O.detect_plane(X, None, P(sigma_mf=0.0, bg_kernel=1, k_bg=K))
        C0 = 2 * math.pi * sig ** 2 * A / (2 * K + 1) ** 2
        assert abs(d["C_last"][40, 40] - C0) / C0 < 2e-4
        m = (A - d["C_last"][40, 40]) / math.sqrt(d["S_last"][40, 40])
        assert abs(m - margin) < 0.2
        assert d["P"].sum() == 1 and d["P"][40, 40] == 1        # isolated noiseless source -> exactly one peak
        assert abs(d["snr"][40, 40] - m) < 1e-12


def test_white_noise_spread_expectation():
    # E[S] = sigma^2 (1 - 2 G00 + sum G^2) for white noise, sigma_mf = 0  (0.9984 for K = 12)
    rng = np.random.default_rng(8)
    X = rng.standard_normal((300, 300)) * 1.7
    for (kind, s, k) in ((1, 0.0, 12), (0, 3.0, 12)):
        g = O.kernel_taps(kind, s, k)
        G = np.outer(g, g)
        want = 1.7 ** 2 * (1 - 2 * G[k, k] + (G ** 2).sum())
        d = O.detect_plane(X, None, P(sigma_mf=0.0, bg_kernel=kind, s_bg=s, k_bg=k, kappa=50.0), direct=False)
        got = d["S_last"][2 * k:-2 * k, 2 * k:-2 * k].mean()
        assert abs(got - want) / want < 0.02
    g = O.kernel_taps(1, 0, 12); G = np.outer(g, g)
    assert abs((1 - 2 * G[12, 12] + (G ** 2).sum()) - 0.9984) < 1e-4


def test_scale_invariance_and_offset():
    s = synth.CubeStream(2)
    X = s.frame(0)[3].astype(np.float64)[:128, :128]
    p = P()
    d0 = O.detect_plane(X, None, p, direct=False)
    assert d0["P"].sum() >= 5
    for a in (2.0, 0.125, 1024.0):
        d = O.detect_plane(a * X, None, p, direct=False)       # power-of-two scale: exact
        assert np.array_equal(d["P"], d0["P"]) and np.array_equal(d["iter"], d0["iter"])
        assert np.allclose(d["snr"], d0["snr"], rtol=1e-12)
    d = O.detect_plane(3.0 * X + 40.0, None, p, direct=False)   # affine: up to rounding
    assert np.array_equal(d["P"], d0["P"])
    assert np.allclose(d["snr"][d0["P"] == 1], d0["snr"][d0["P"] == 1], rtol=1e-9)


def test_eps_rel_guard_only_acts_on_rounding_noise():
    # S_eff = max(S, (eps |C|)^2): a huge offset on a tiny-noise image silences detections (R8)
    rng = np.random.default_rng(9)
    X = 1e9 + rng.standard_normal((64, 64)) * 1.0
    X[30, 30] += 8.0
    d = O.detect_plane(X, None, P(sigma_mf=0.0))
    assert d["P"].sum() == 0                     # sqrt(S) ~ 1 << eps_rel * 1e9 = 1e4
    d = O.detect_plane(X - 1e9, None, P(sigma_mf=0.0))
    assert d["P"][30, 30] == 1


def test_deblending():
    # two noiseless sources (10 and 7): 4 px apart -> two peaks at their pixels; 3 px -> one
    for bg in (dict(bg_kernel=1, k_bg=12), dict(bg_kernel=0, s_bg=8.0, k_bg=16)):
        for sep, want in ((4, 2), (3, 1)):
            X = gauss_img(81, 40, 38, 10.0, SIG) + gauss_img(81, 40, 38 + sep, 7.0, SIG)
            d = O.detect_plane(X, None, P(**bg))
            assert d["P"].sum() == want, (bg, sep)
            assert d["P"][40, 38] == 1
            if want == 2:
                assert d["P"][40, 38 + sep] == 1


def test_sigma_clip_iterations_accumulate():
    # a faint source next to a bright one is found only once the bright one is clipped away
    rng = np.random.default_rng(10)
    X = rng.standard_normal((96, 96)) * 0.05
    X += gauss_img(96, 48, 40, 40.0, 1.5)      # bright: inflates S around it
    X += gauss_img(96, 48, 50, 4.0, SIG)       # faint neighbour inside the bright one's window
    p1 = P(n_iter=1, sigma_mf=0.0, k_max=2)
    p3 = P(n_iter=6, sigma_mf=0.0, k_max=2)
    d1 = O.detect_plane(X, None, p1); d3 = O.detect_plane(X, None, p3)
    assert d1["P"][48, 40] == 1 and d1["P"][48, 50] == 0
    assert d3["P"][48, 40] == 1 and d3["P"][48, 50] == 1 and d3["iter"][48, 50] > 1
    assert np.all(d3["iter"][d1["iter"] > 0] == 1)          # Y accumulates; first-iteration pixels keep iter = 1
    # "pre-specified number of iterations" beyond convergence changes nothing
    d9 = O.detect_plane(X, None, P(n_iter=60, sigma_mf=0.0))
    d8 = O.detect_plane(X, None, P(n_iter=40, sigma_mf=0.0))
    assert np.array_equal(d9["iter"], d8["iter"])


def test_false_negative_law_eq1():
    # PAPER.md:55 eq. 1: Pr(FN) = Phi(kappa - s/n)^B, paper-literal mode (sigma_mf = 0, single-pixel source)
    rng = np.random.default_rng(11)
    kappa, D = 3.0, 290
    p = P(kappa=kappa, sigma_mf=0.0, k_max=2, bg_kernel=1, k_bg=12)
    ys, xs = np.meshgrid(np.arange(20, 270, 26), np.arange(20, 270, 26), indexing="ij")  # one source per window
    ys, xs = ys.ravel(), xs.ravel()
    for snr, B in ((2.0, 1), (3.0, 1), (4.0, 1), (3.0, 4)):
        miss = tot = 0
        for trial in range(6):
            hit = np.zeros(ys.size, bool)
            for b in range(B):
                X = rng.standard_normal((D, D))
                X[ys, xs] += snr
                Y = O.detect_plane(X, None, p, direct=False)["iter"] > 0   # eq. 5 is about y_nm
                hit |= Y[ys, xs]
            miss += (~hit).sum(); tot += ys.size
        want = sst.norm.cdf(kappa - snr) ** B
        assert abs(miss / tot - want) < 0.05, (snr, B, miss / tot, want)


# ---------------------------------------------------------------- O6 ---------
def test_local_max_equals_scipy_maximum_filter():
    rng = np.random.default_rng(12)
    X = rng.standard_normal((50, 63))
    X[10, 10] = X[10, 11] = 9.0     # a plateau: both are maxima (equality form, reading R9)
    for k in (1, 2, 3):
        d = O.detect_plane(X, None, P(sigma_mf=0.0, k_max=k, kappa=1.0))
        ref = X == ndi.maximum_filter(X, size=2 * k + 1, mode="constant", cval=-np.inf)
        assert np.array_equal(d["Q"].astype(bool), ref)
        assert np.array_equal(d["P"].astype(bool), ref & (d["iter"] > 0))   # eq. 7
    assert d["Q"][10, 10] == 1 and d["Q"][10, 11] == 1
    # masked pixels are skipped by the window and are never maxima
    W = (rng.random((50, 63)) > 0.3).astype(np.uint8)
    d = O.detect_plane(X, W, P(sigma_mf=0.0, k_max=2, kappa=1.0))
    Xm = np.where(W == 1, d["F"], -np.inf)
    ref = (Xm == ndi.maximum_filter(Xm, size=5, mode="constant", cval=-np.inf)) & (W == 1)
    assert np.array_equal(d["Q"].astype(bool), ref)


# ------------------------------------------------------- whole chain, brute --
def _brute_plane(X, W, g_mf, g_bg, kappa, eps, n_iter, k_max):
    """Independent pure-Python evaluation of eqs. 2-7 with 4 nested loops (tiny inputs only)."""
    Dy, Dx = X.shape

    def nconv(A, Wp, g):
        k = (len(g) - 1) // 2
        out = np.zeros_like(A)
        for n in range(Dy):
            for m in range(Dx):
                num = den = 0.0
                for i in range(max(0, n - k), min(Dy, n + k + 1)):
                    for j in range(max(0, m - k), min(Dx, m + k + 1)):
                        if Wp[i, j]:
                            w = g[i - n + k] * g[j - m + k]
                            num += w * A[i, j]; den += w
                out[n, m] = num / den if den > 0 else 0.0
        return out

    F = nconv(X, W, g_mf) * (W > 0)
    Y = np.zeros((Dy, Dx), int)
    for it in range(1, n_iter + 1):
        Wp = (W > 0) & (Y == 0)
        Cc = nconv(F, Wp, g_bg)
        S = nconv((F - Cc) ** 2, Wp, g_bg)
        Se = np.maximum(S, (eps * np.abs(Cc)) ** 2)
        new = (Y == 0) & (W > 0) & (F - Cc > 0) & ((F - Cc) ** 2 > kappa ** 2 * Se)
        Y[new] = it
    Pk = np.zeros((Dy, Dx), int)
    for n in range(Dy):
        for m in range(Dx):
            if not W[n, m] or not Y[n, m]:
                continue
            mx = max(F[i, j] for i in range(max(0, n - k_max), min(Dy, n + k_max + 1))
                     for j in range(max(0, m - k_max), min(Dx, m + k_max + 1)) if W[i, j])
            Pk[n, m] = int(F[n, m] == mx)
    return F, Y, Pk


@pytest.mark.parametrize("bg", ["box", "gauss"])
def test_whole_plane_brute_force_tiny(bg):
    rng = np.random.default_rng(13)
    Dy, Dx = 24, 29
    X = rng.standard_normal((Dy, Dx))
    X += gauss_img(40, 9, 12, 12.0, SIG)[:Dy, :Dx] + gauss_img(40, 17, 22, 8.0, SIG)[:Dy, :Dx]
    W = np.ones((Dy, Dx), np.uint8); W[0:5, 0:6] = 0; W[12, 14] = 0
    kw = dict(bg_kernel=1, k_bg=4) if bg == "box" else dict(bg_kernel=0, s_bg=2.5, k_bg=5)
    p = P(kappa=3.0 if bg == "box" else 2.2, n_iter=3, k_mf=2, **kw)
    g_mf = O.kernel_taps(0, p["sigma_mf"], p["k_mf"]); g_bg = O.kernel_taps(p["bg_kernel"], p["s_bg"], p["k_bg"])
    F, Y, Pk = _brute_plane(X, W, g_mf, g_bg, p["kappa"], p["eps_rel"], p["n_iter"], p["k_max"])
    for direct in (True, False):
        d = O.detect_plane(X, W, p, direct=direct)
        assert np.allclose(d["F"], F, rtol=1e-12, atol=1e-14)
        assert np.array_equal(d["iter"], Y) and np.array_equal(d["P"], Pk)
    assert Pk.sum() >= 2 and (Y > 1).any()


def test_config1_whole_chain():
    # config 1: the 10 sigma source is a peak at (y,x) = (20,37) in all 4 channel planes and the sum plane in
    # every frame (SURVEY 8(c) "whole chain").  Anything else is a >5 sigma noise excursion: with this seed
    # there is exactly one in 32 frames x 5 planes x 4096 px (frame 22, plane 3, snr 5.05).
    s = synth.CubeStream(1)
    src = 20 * 64 + 37
    for bg, n_iter in (("box", 1), ("gauss", 1), ("box", 3)):
        p = synth.default_params(1, bg=bg, n_iter=n_iter)
        full = (bg == "box" and n_iter == 1)
        pipe = O.OraclePipeline(p, s.mask, direct=full)
        n_other = 0
        for t in range(32 if full else 6):
            r = pipe.step(s.frame(t), t)
            assert r["band_ok"].all()
            assert src in r["upos"].tolist()
            at_src = r["rec"][r["rec"]["pix"] == src]
            assert sorted(at_src["plane"].tolist()) == [0, 1, 2, 3, 4]
            other = r["rec"][r["rec"]["pix"] != src]
            n_other += other.size
            assert (other["snr"] < 5.5).all()
            i = r["upos"].tolist().index(src)
            assert r["cand_idx"][i] == 0 and r["act_slots"][0] == 0 and r["act_pix"][0] == src
            # forced flux at the source: 10 sigma peak + noise, same pixel box in every band
            assert r["flux"].shape[1] == 4 and (r["flux"][0] > 6).all()
        assert n_other <= 1
        ds = pipe.table.dynspec(0)
        assert ds.shape == (4, p["T_ring"]) and np.isfinite(ds[:, -1]).all()


# ---------------------------------------------------------------- O7 / O8 ----
def test_dedupe_rules_and_order_independence():
    Dx = Dy = 100
    pix = np.array([10 * Dx + 10, 10 * Dx + 10, 10 * Dx + 12, 11 * Dx + 11, 50 * Dx + 50, 50 * Dx + 53, 70 * Dx + 70, 70 * Dx + 72])
    plane = np.array([0, 3, 1, 2, 0, 1, 4, 5], np.int16)
    snr = np.array([6.0, 9.0, 8.0, 7.0, 6.0, 6.5, 7.0, 7.0])
    up, upl, us = O.dedupe(pix, plane, snr, Dy, Dx, 2)
    # (10,10): M = 9 from plane 3 beats (10,12) [d=2] and (11,11); (50,50)/(50,53): d=3 > r -> both kept;
    # (70,70) vs (70,72): equal M -> lower pix wins
    assert up.tolist() == [10 * Dx + 10, 50 * Dx + 50, 50 * Dx + 53, 70 * Dx + 70]
    assert upl.tolist() == [3, 0, 1, 4] and us.tolist() == [9.0, 6.0, 6.5, 7.0]
    rng = np.random.default_rng(14)
    for _ in range(5):
        perm = rng.permutation(pix.size)
        up2, upl2, us2 = O.dedupe(pix[perm], plane[perm], snr[perm], Dy, Dx, 2)
        assert up2.tolist() == up.tolist() and upl2.tolist() == upl.tolist() and us2.tolist() == us.tolist()
    # equal snr at one pixel -> lowest plane
    _, upl3, _ = O.dedupe(np.array([5, 5]), np.array([7, 2], np.int16), np.array([6.0, 6.0]), Dy, Dx, 2)
    assert upl3.tolist() == [2]
    # one-shot suppression (not greedy): chain a<b<c with d(a,b), d(b,c) <= r: only c survives
    up4, _, _ = O.dedupe(np.array([0, 2, 4]), np.zeros(3, np.int16), np.array([5.0, 6.0, 7.0]), Dy, Dx, 2)
    assert up4.tolist() == [4]
    assert O.dedupe(np.zeros(0), np.zeros(0), np.zeros(0), Dy, Dx, 2)[0].size == 0


def test_association_monitoring_and_slots():
    Dx = 100
    tb = O.CandidateTable(8, 4, 2, Dx, r_assoc=3, n_forget=2)
    a, b, c = 10 * Dx + 10, 40 * Dx + 40, 70 * Dx + 70
    cand, s, p = tb.associate(np.array([a, b]), 0, 1)
    assert cand.tolist() == [0, 1] and s.tolist() == [0, 1] and p.tolist() == [a, b]
    # idempotence: the same frame again creates no new slots
    cand, s, p = tb.associate(np.array([a, b]), 1, 1)
    assert cand.tolist() == [0, 1] and s.tolist() == [0, 1]
    # jittered detection within r_assoc matches; candidate keeps its first pixel; d^2 = 9 is inside, 10 is not
    cand, s, p = tb.associate(np.array([a + 3, b + 3 * Dx + 1]), 2, 1)
    assert cand.tolist() == [0, 2] and p.tolist() == [a, b, b + 3 * Dx + 1]
    # rejected frame: nothing changes, detections unassigned
    miss_before = tb.miss.copy()
    cand, s, p = tb.associate(np.array([c]), 3, 0)
    assert cand.tolist() == [-1] and np.array_equal(tb.miss, miss_before) and s.tolist() == [0, 1, 2]
    # slot 1 missed at t=2 (miss 1); missing again -> retired at n_forget = 2; c takes the lowest free slot (1)
    cand, s, p = tb.associate(np.array([a, c]), 4, 1)
    assert cand.tolist() == [0, 1] and s.tolist() == [0, 1, 2] and p.tolist() == [a, c, b + 3 * Dx + 1]
    # nearest wins; equal distance -> lowest slot
    tb2 = O.CandidateTable(8, 4, 2, Dx, 3, 5)
    tb2.associate(np.array([20 * Dx + 20, 20 * Dx + 24]), 0, 1)
    cand, _, _ = tb2.associate(np.array([20 * Dx + 22, 20 * Dx + 23]), 1, 1)
    assert cand.tolist() == [0, 1]
    # forced candidates are never retired; capacity overflow drops and counts
    tb3 = O.CandidateTable(3, 4, 2, Dx, 3, 1)
    tb3.add_forced(np.array([a]))
    for t in range(4):
        tb3.associate(np.array([], np.int32), t, 1)
    assert tb3.active.tolist() == [1, 0, 0]
    cand, s, _ = tb3.associate(np.array([b, c, 90 * Dx + 90]), 5, 1)
    assert cand.tolist() == [1, 2, -1] and int(tb3.n_dropped[0]) == 1
    # order independence of the result w.r.t. candidate/detection content is by construction: detections arrive
    # sorted by pix from dedupe; matching uses only the pre-frame table (two new detections within r_assoc of
    # each other both get slots)
    tb4 = O.CandidateTable(8, 4, 2, Dx, 3, 5)
    cand, _, _ = tb4.associate(np.array([5 * Dx + 5, 5 * Dx + 8]), 0, 1)
    assert cand.tolist() == [0, 1]


# ---------------------------------------------------------------- O9 / O10 ---
def test_forced_flux():
    D, B = 40, 3
    A = np.float32(12.3456789)
    cube = np.zeros((B, D, D), np.float32)
    cube[:, 20, 21] = A          # noiseless injected source, integer-pixel centre
    cube[1, 20, 21] = -A
    cube[2, 19, 20] = 2 * A
    ok = np.ones(B + 1, np.uint8)
    f = O.measure_flux(cube, ok, None, np.array([20 * D + 21, 20 * D + 20, 0, D * D - 1]), 1)
    assert f[0].tolist() == [A, 0.0, 2 * A]            # exact; band 1: max of (-A, zeros) = 0
    assert f[1].tolist() == [A, 0.0, 2 * A]            # within +-1 px the peak is still inside the box
    assert f[2].tolist() == [0, 0, 0] and f[3].tolist() == [0, 0, 0]   # corners: in-image part only
    # maximum, not sum / mean; negative field -> largest value
    cube2 = -np.ones((1, 5, 5), np.float32); cube2[0, 2, 2] = -0.5
    assert O.measure_flux(cube2, np.ones(2, np.uint8), None, np.array([12]), 1)[0, 0] == np.float32(-0.5)
    # rejected band -> 0 ; rejected frame -> all 0 ; masked pixels skipped
    ok2 = np.array([1, 0, 1, 1], np.uint8)
    assert O.measure_flux(cube, ok2, None, np.array([20 * D + 21]), 1)[0].tolist() == [A, 0.0, 2 * A]
    ok3 = np.array([1, 1, 1, 0], np.uint8)
    assert O.measure_flux(cube, ok3, None, np.array([20 * D + 21]), 1)[0].tolist() == [0, 0, 0]
    W = np.ones((D, D), np.uint8); W[19, 20] = 0
    assert O.measure_flux(cube, ok, W, np.array([20 * D + 21]), 1)[0].tolist() == [A, 0.0, A]
    # unit noise: mean of the max of 9 standard normals = 1.4850
    rng = np.random.default_rng(15)
    noise = rng.standard_normal((1, 300, 300)).astype(np.float32)
    pos = (np.arange(10, 290, 3)[:, None] * 300 + np.arange(10, 290, 3)[None, :]).ravel()
    fl = O.measure_flux(noise, np.ones(2, np.uint8), None, pos, 1)
    assert abs(fl.mean() - 1.4850) < 0.02
    # r_flux = 2 box
    assert O.measure_flux(cube, ok, None, np.array([22 * D + 23]), 2)[0].tolist() == [A, 0.0, A]


def test_ring_buffer_wraparound_and_view():
    T, B = 8, 3
    tb = O.CandidateTable(4, T, B, 100, 3, 100)
    ok = np.ones(B + 1, np.uint8)
    tb.associate(np.array([555]), 0, 1)
    assert np.isnan(tb.dynspec(0, 0)).all()                 # new slot reads NaN before the first append
    for t in range(T + 3):
        if t == 5:
            tb.associate(np.array([555, 5555]), t, 1)       # second candidate born at t = 5
        slots = np.flatnonzero(tb.active).astype(np.int32)
        flux = np.array([[100 * s + t + 0.1 * b for b in range(B)] for s in slots], np.float32)
        okt = ok.copy()
        if t == 7:
            okt[1] = 0
        tb.append(slots, flux, okt, t)
    ds = tb.dynspec(0)
    # after T+3 appends the 3 oldest samples are gone; columns are time ordered, oldest -> newest
    assert np.allclose(ds[0], np.arange(3, T + 3), atol=1e-6)
    assert np.allclose(ds[2], np.arange(3, T + 3) + 0.2, atol=1e-5)
    ds1 = tb.dynspec(1)
    assert np.isnan(ds1[:, :2]).all() and np.allclose(ds1[0, 2:], 100 + np.arange(5, T + 3), atol=1e-5)
    assert int(tb.meta_ok[7 % T]) == 0b101 and int(tb.meta_ok[8 % T]) == 0b111
    assert tb.meta_t.tolist() == [8, 9, 10, 3, 4, 5, 6, 7]


# ------------------------------------------------- injected sources recovered -
def test_injected_sources_recovered_config2():
    # north_star pin: injected sources of known position and flux are recovered.
    s = synth.CubeStream(2)
    p = synth.default_params(2)
    pipe = O.OraclePipeline(p, s.mask, direct=False)
    r = pipe.step(s.frame(0), 0)
    D = 256
    uy, ux = r["upos"] // D, r["upos"] % D
    st = s.steady
    iso = []
    for i in range(st["y"].size):     # isolated bright sources away from the border
        d2 = (st["y"] - st["y"][i]) ** 2 + (st["x"] - st["x"][i]) ** 2
        d2[i] = 10 ** 9
        if st["snr"][i] >= 9 and d2.min() > 15 ** 2 and 15 <= st["y"][i] < D - 15 and 15 <= st["x"][i] < D - 15:
            iso.append(i)
    assert len(iso) >= 8
    for i in iso:
        d2 = (uy - st["y"][i]) ** 2 + (ux - st["x"][i]) ** 2
        j = int(np.argmin(d2))
        assert d2[j] <= 1, (i, st["snr"][i])                       # position recovered to +-1 px
        k = r["act_pix"].tolist().index(int(r["upos"][j]))
        fl = r["flux"][k]                                           # forced flux ~ amplitude (+ max-of-9 noise bias)
        assert abs(np.median(fl) - st["amp"][i]) < 1.5
    assert r["upos"].size < 1.5 * st["y"].size                      # and not swamped by false positives


# ------------------------------------------------------------------ O11 backward fill
def _ramp_stream(n_frames=14, D=64, B=4, seed=3):
    rng = np.random.default_rng(seed)
    yy, xx = np.mgrid[0:D, 0:D]
    g = np.exp(-0.5 * ((yy - 30) ** 2 + (xx - 41) ** 2) / 0.85 ** 2).astype(np.float32)
    amp = [0, 0, 0, 0, 0, 1.5, 2.5, 3.5, 4.5, 6.0, 9.0, 14.0, 20.0, 20.0]
    return [(rng.standard_normal((B, D, D)).astype(np.float32) + amp[t] * g) for t in range(n_frames)]


def test_backward_fill_shows_the_build_up():
    """A source that brightens slowly is first detected at t_d; with n_back = 4 its dynamic spectrum must then
    hold, for t_d-4 .. t_d-1, the box maximum of those EARLIER cubes at its pixel (computed here with plain
    NumPy slicing), NaN before that, and the ordinary monitored fluxes from t_d on.  n_back = 0: NaN before t_d."""
    import oracle as O
    from paper_2103_15418_b200 import synth
    cubes = _ramp_stream()
    B, D, _ = cubes[0].shape
    p = synth.default_params(1); p.update(B=B, Dy=D, Dx=D, T_ring=16)
    res = {}
    for nb in (0, 4):
        q = dict(p); q["n_back"] = nb
        pipe = O.OraclePipeline(q, None, direct=False)
        for t, c in enumerate(cubes):
            pipe.step(c, t)
        tb = pipe.table
        slots = [s for s in np.flatnonzero(tb.active) if abs(tb.cpix[s] // D - 30) <= 1 and abs(tb.cpix[s] % D - 41) <= 1]
        assert len(slots) == 1
        s = slots[0]
        res[nb] = (int(tb.born[s]), int(tb.cpix[s]), pipe.table.dynspec(int(s), len(cubes) - 1))
    t_d, pix, ds0 = res[0]
    assert res[4][0] == t_d and res[4][1] == pix and 5 < t_d < 12
    y, x = divmod(pix, D)
    T = 16
    col = lambda t: T - 1 - (len(cubes) - 1 - t)          # dynspec is time ordered, newest last
    ds4 = res[4][2]
    for t in range(len(cubes)):
        want = np.array([cubes[t][b, y - 1:y + 2, x - 1:x + 2].max() for b in range(B)], np.float32)
        if t >= t_d:                                        # monitored from birth on, with or without backfill
            assert np.array_equal(ds0[:, col(t)], want) and np.array_equal(ds4[:, col(t)], want)
        else:
            assert np.isnan(ds0[:, col(t)]).all()
            if t >= t_d - 4:
                assert np.array_equal(ds4[:, col(t)], want), t
            else:
                assert np.isnan(ds4[:, col(t)]).all()


def test_backward_fill_respects_rejected_bands_and_ring_age():
    import oracle as O
    from paper_2103_15418_b200 import synth
    cubes = _ramp_stream()
    B, D, _ = cubes[0].shape

    def run(T_ring, n_back, nan_at=None):
        p = synth.default_params(1); p.update(B=B, Dy=D, Dx=D, T_ring=T_ring, n_back=n_back)
        pipe = O.OraclePipeline(p, None, direct=False)
        for t, c in enumerate(cubes):
            c = c.copy()
            if nan_at is not None and t == nan_at:
                c[2, 0, 0] = np.nan              # band 2 is rejected in that frame (non-finite statistics)
            pipe.step(c, t)
            tb = pipe.table
            hit = [s for s in np.flatnonzero(tb.active) if abs(tb.cpix[s] // D - 30) <= 1 and abs(tb.cpix[s] % D - 41) <= 1]
            if hit:
                return t, int(tb.cpix[hit[0]]), tb.ring[int(hit[0])].copy(), tb.meta_t.copy()
        raise AssertionError("never detected")

    t_d, pix, _, _ = run(16, 4)
    y, x = divmod(pix, D)
    # a band rejected in a cached frame: its back-filled flux is 0, the other bands are the box maxima
    t2, pix2, ring, meta = run(16, 4, nan_at=t_d - 2)
    assert (t2, pix2) == (t_d, pix)
    colv = ring[(t_d - 2) % 16]
    assert colv[2] == 0.0
    for b in (0, 1, 3):
        assert colv[b] == cubes[t_d - 2][b, y - 1:y + 2, x - 1:x + 2].max()
    # a ring shorter than the cache: only columns that still belong to their frame are filled
    t3, pix3, ring, meta = run(3, 6)
    assert (t3, pix3) == (t_d, pix)
    assert sorted(meta.tolist()) == [t_d - 2, t_d - 1, t_d]
    for tau in (t_d - 2, t_d - 1, t_d):
        want = np.array([cubes[tau][b, y - 1:y + 2, x - 1:x + 2].max() for b in range(B)], np.float32)
        assert np.array_equal(ring[tau % 3], want)


# ------------------------------------------------------------------ O12 running per-pixel QC (eq. A.2)
def test_running_qc_is_welford_then_exponential():
    import oracle as O
    rng = np.random.default_rng(11)
    B, D, Nw = 2, 8, 16
    rq = O.RunningQC(B, D, D, thr=1e9, nmax=0, window=Nw, warm=4)
    frames = [(3.0 + 2.0 * rng.standard_normal((B, D, D))).astype(np.float32) for _ in range(Nw)]
    ok = np.ones(B + 1, np.uint8)
    for k, f in enumerate(frames):
        cnt, ok2 = rq.step(f, None, ok)
        assert ok2.all() and not cnt.any()
        st = np.stack(frames[:k + 1]).astype(np.float64)
        # Welford (1962): after k+1 <= window updates the state IS the sample mean and the population variance
        assert np.allclose(rq.m, st.mean(0), rtol=2e-6, atol=2e-6)
        assert np.allclose(rq.v, st.var(0), rtol=2e-5, atol=2e-6)
    assert (rq.n == Nw).all()
    # Finch (2009): from here on alpha = 1/window; a step of height h is followed as h (1 - (1 - alpha)^k)
    base = rq.m.copy()
    h = np.float32(5.0)
    for k in range(1, 9):
        rq.step(base + h, None, ok)
        assert np.allclose(rq.m - base, h * (1.0 - (1.0 - 1.0 / Nw) ** k), rtol=1e-5, atol=1e-5)


def test_running_qc_verdict_rules():
    import oracle as O
    rng = np.random.default_rng(12)
    B, D = 4, 16
    W = np.ones((D, D), np.uint8); W[0, :] = 0
    mk = lambda: rng.standard_normal((B, D, D)).astype(np.float32)
    rq = O.RunningQC(B, D, D, thr=15.0, nmax=0, window=32, warm=8)
    ok = np.ones(B + 1, np.uint8)
    for t in range(8):
        f = mk()
        if t == 3:
            f[1, 5, 5] = 1e4                      # before the warm-up is over nothing is tested
        cnt, o = rq.step(f, W, ok)
        assert o.all() and not cnt.any()
    for _ in range(20):
        rq.step(mk(), W, ok)                      # let the spike of t = 3 decay out of band 1's variance
    f = mk(); f[2, 7, 9] += 200.0; f[3, 0, 4] += 200.0      # a spike at a valid pixel, one at a masked pixel
    before = (rq.m.copy(), rq.v.copy(), rq.n.copy())
    cnt, o = rq.step(f, W, ok)
    assert cnt.tolist() == [0, 0, 1, 0] and o.tolist() == [1, 1, 0, 1, 1]
    # the discarded band keeps its state (test before update, update only accepted bands); the others moved on
    assert np.array_equal(rq.m[2], before[0][2]) and np.array_equal(rq.v[2], before[1][2]) and rq.n[2] == before[2][2]
    assert not np.array_equal(rq.m[0], before[0][0]) and rq.n[0] == before[2][0] + 1
    # count rule: with nmax = 1 the same frame passes; bands rejected by eq. A.1 are neither tested away nor updated
    rq2 = O.RunningQC(B, D, D, thr=15.0, nmax=1, window=32, warm=8)
    for _ in range(10):
        rq2.step(mk(), W, ok)
    f = mk(); f[2, 7, 9] += 200.0
    cnt, o = rq2.step(f, W, ok)
    assert cnt[2] == 1 and o.all()
    a1 = np.array([1, 0, 0, 1, 1], np.uint8)     # two bands already rejected by eq. A.1
    n0 = rq2.n.copy()
    cnt, o = rq2.step(mk(), W, a1)
    assert o.tolist() == [1, 0, 0, 1, 1] and (rq2.n - n0).tolist() == [1, 0, 0, 1]
    f = mk(); f[0, 3, 3] += 500.0
    cnt, o = rq2.step(f, W, a1)                   # one spike: passes (nmax = 1)
    assert o[0] == 1
    f = mk(); f[0, 8, 8] += 500.0; f[0, 9, 2] += 500.0
    cnt, o = rq2.step(f, W, a1)
    assert cnt[0] == 2 and o.tolist() == [0, 0, 0, 1, 0]       # one accepted band of four: the frame is rejected


def test_running_qc_variance_recurrence_and_stationary_value():
    """eq. A.2 + R22 written out here in plain float64 NumPy, per pixel, through the Welford phase and far into the
    exponentially weighted phase: m += a d, v = (1 - a)(v + a d^2), a = 1/min(k, window).  The oracle (float32 state,
    one rounding per update) must follow it; and for a stationary stream of variance s^2 the recurrence has the
    closed-form expectations  E[d^2] = 2 s^2/(2 - a),  E[v] = (1 - a) 2 s^2/(2 - a)  (k >> window)."""
    import oracle as O
    rng = np.random.default_rng(13)
    B, D, Nw, sig = 2, 48, 16, 2.5
    rq = O.RunningQC(B, D, D, thr=1e9, nmax=0, window=Nw, warm=4)
    ok = np.ones(B + 1, np.uint8)
    m = np.zeros((B, D, D)); v = np.zeros((B, D, D))
    vs = []
    for k in range(1, 12 * Nw + 1):
        x = (1.0 + sig * rng.standard_normal((B, D, D))).astype(np.float32)
        rq.step(x, None, ok)
        a = 1.0 / min(k, Nw)
        d = x.astype(np.float64) - m
        m = m + a * d
        v = (1.0 - a) * (v + a * d * d)
        if k in (3, Nw, Nw + 1, 2 * Nw, 12 * Nw):
            assert np.allclose(rq.m, m, rtol=0, atol=3e-5 * sig), k          # float32 state, contractive recurrence
            assert np.allclose(rq.v, v, rtol=3e-5, atol=1e-6), k
        if k > 6 * Nw:
            vs.append(rq.v.astype(np.float64).mean())
    a = 1.0 / Nw
    want = (1.0 - a) * 2.0 * sig ** 2 / (2.0 - a)                             # 0.9677 s^2 for window 16
    assert abs(np.mean(vs) / want - 1.0) < 0.01, (np.mean(vs), want)
    # the nearest wrong recurrences are 3-7 % away: v = (1-a) v + a d^2 gives 2 s^2/(2-a); plain s^2 is 1.000
    assert abs(np.mean(vs) / (2.0 * sig ** 2 / (2.0 - a)) - 1.0) > 0.04 and abs(np.mean(vs) / sig ** 2 - 1.0) > 0.02


def test_running_qc_zeta_threshold_edge_and_zero_variance():
    """|zeta| = thr (1 +- 1e-3): after the two frames +1, -1 the state is m = 0, v = 1 exactly (Welford), so a pixel
    at thr (1 + 1e-3) exceeds and one at thr (1 - 1e-3) does not, either sign; a pixel whose stream was constant so far
    (v = 0) has no zeta and is not counted."""
    import oracle as O
    B, D, thr = 1, 8, 15.0
    rq = O.RunningQC(B, D, D, thr=thr, nmax=0, window=64, warm=2)
    ok = np.ones(B + 1, np.uint8)
    f = np.ones((B, D, D), np.float32); f[0, 7, 7] = 0.0
    g = -f
    rq.step(f, None, ok); rq.step(g, None, ok)
    assert np.array_equal(rq.m[0, :7, :7], np.zeros((7, 7), np.float32)) and np.array_equal(rq.v[0, :7, :7], np.ones((7, 7), np.float32))
    assert rq.v[0, 7, 7] == 0.0
    x = np.zeros((B, D, D), np.float32)
    x[0, 1, 1] = thr * (1 + 1e-3); x[0, 2, 2] = thr * (1 - 1e-3); x[0, 3, 3] = -thr * (1 + 1e-3); x[0, 4, 4] = -thr * (1 - 1e-3)
    x[0, 7, 7] = 1e6                                     # v = 0 there: not tested
    cnt, o = rq.step(x, None, ok)
    assert cnt.tolist() == [2] and o.tolist() == [0, 0]
    rq2 = O.RunningQC(B, D, D, thr=thr, nmax=2, window=64, warm=2)
    rq2.step(f, None, ok); rq2.step(g, None, ok)
    cnt, o = rq2.step(x, None, ok)
    assert cnt.tolist() == [2] and o.tolist() == [1, 1]      # count rule: 2 > 2 is false
    W = np.ones((D, D), np.uint8); W[1, 1] = 0
    rq3 = O.RunningQC(B, D, D, thr=thr, nmax=0, window=64, warm=2)
    rq3.step(f, W, ok); rq3.step(g, W, ok)
    assert rq3.step(x, W, ok)[0].tolist() == [1]             # the masked one does not count


def test_running_qc_recovers_after_a_lasting_level_change():
    """R22: a band discarded by eq. A.2 keeps its state, so after a lasting level change it would stay discarded for
    good; with zeta_reset = 3 it starts over after three consecutive discards and is accepted again after the warm-up."""
    import oracle as O
    rng = np.random.default_rng(14)
    B, D = 2, 16
    mk = lambda off: (off + rng.standard_normal((B, D, D))).astype(np.float32)
    ok = np.ones(B + 1, np.uint8)
    for reset, want_back in ((0, False), (3, True)):
        rq = O.RunningQC(B, D, D, thr=8.0, nmax=4, window=16, warm=4, reset=reset)
        for _ in range(12):
            assert rq.step(mk(0.0), None, ok)[1].all()
        verdicts = []
        for k in range(12):
            f = mk(0.0); f[1] += 100.0                   # band 1 jumps by 100 sigma and stays there
            verdicts.append(int(rq.step(f, None, ok)[1][1]))
        if want_back:
            assert verdicts[:3] == [0, 0, 0] and all(verdicts[3:]), verdicts      # reset after the 3rd, untested warm-up, then fine
            assert abs(float(rq.m[1].mean()) - 100.0) < 1.0
        else:
            assert not any(verdicts)


# ------------------------------------------------------------------ O13 / O14 network input and simulated pulses
def test_simulated_pulse_closed_forms():
    """eqs. 19-21: the peak of band nu sits at t0 + delay(nu) with the golden delays of eq. 20, its height is
    A (nu/nu0)^alpha, the full width at half maximum is 2 sqrt(2 ln 2) w (w = 16 <-> 37.67, :197-199), DM = 0 is
    undispersed."""
    import oracle as O
    nu = np.array([57.0, 58.3671875, 61.7, 63.0671875]); nu0 = 63.1
    T = 4096
    th = np.array([[300.0, 16.0, 30.0, 5.0, -2.0], [900.25, 40.0, 0.0, 2.0, 1.5]])
    I = O.simulate_pulses(th, nu, nu0, T, dt=0.01)            # 10 ms steps: the delays span hundreds of steps
    gold = {57.0: 7.0487, 58.3671875: 5.2750, 61.7: 1.4347, 63.0671875: 0.0325}   # s, tests/golden/dispersion_delays.txt
    for b, v in enumerate(nu):
        tp = int(np.argmax(I[0, b]))
        assert abs(tp - (300.0 + gold[v] / 0.01)) <= 1.0
        assert np.isclose(I[0, b].max(), 5.0 * (v / nu0) ** -2.0, rtol=2e-3)
        above = np.flatnonzero(I[0, b] >= 0.5 * I[0, b].max())
        assert abs((above[-1] - above[0]) - 37.67) <= 2.0        # sampled at integer steps
        assert int(np.argmax(I[1, b])) == 900 and np.isclose(I[1, b, 900], 2.0 * (v / nu0) ** 1.5 * np.exp(-0.5 * (0.25 / 40) ** 2))
    assert np.isclose(O.C_DM * (1000.0 ** -2), 4.148806e-3)   # 4.1488 ms at 1 GHz for DM = 1 (:206)


def test_export_dynspec_is_the_ordered_normalised_view():
    import oracle as O
    tb = O.CandidateTable(8, 6, 3, 16, 3, 10)
    slots = tb.add_forced(np.array([5, 40], np.int32))
    ok = np.ones(4, np.uint8)
    for t in range(9):                                         # more frames than the ring holds
        flux = np.array([[t + 0.0, 10 * t + 1.0, 100 * t + 2.0], [-t, -2.0 * t, -3.0 * t]], np.float32)
        tb.append(slots, flux, ok, t)
    x = O.export_dynspec(tb, slots, 8, sigma=[1.0, 2.0, 0.0])
    assert x.shape == (2, 3, 6) and x.dtype == np.float32
    ts = np.arange(3, 9)                                       # the six newest frames, oldest first
    assert np.array_equal(x[0, 0], ts) and np.allclose(x[0, 1], (10 * ts + 1) / 2.0) and np.array_equal(x[0, 2], 100 * ts + 2)
    assert np.array_equal(x[1, 0], -ts)
    y = O.export_dynspec(tb, slots, 10, sigma=None)            # two frames that do not exist yet: zeros, not NaN
    assert np.array_equal(y[0, 0], [5, 6, 7, 8, 0, 0])
