"""Pins of the CPU oracle (oracle/nfs_oracle.c) against things that are not itself.

Pin numbers are those of SURVEY.md §8(c) / DESIGN.md §3.  All CPU-only (`-m "not gpu"`).
Every pin is chosen so that a plausible mistake (dropped term, wrong sign/index, transposed
axes, wrong divisor, wrong scale) fails at least one of them.
"""
import math
import os

import numpy as np
import pytest

from oracle import brute_force as bf

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "p13_golden.txt")


def _rng(seed):
    return np.random.default_rng(seed)


# ---- P1: DFT / FFT -------------------------------------------------------------------------
def test_p1_bruteforce_dft_8x8_vs_python_loops(oracle):
    img = _rng(1).uniform(0, 10, (8, 8))
    F_c = oracle.transform_f64(img, method=1)          # C brute force
    F_py = np.array(bf.dft2_unitary(img.tolist()))     # pure-Python O(n^4)
    assert np.max(np.abs(F_c - F_py)) < 1e-12


def test_p1_radix2_vs_direct_and_numpy(oracle):
    # non-square on purpose: catches transposed axes
    img = _rng(2).normal(0, 1, (32, 16))
    F_fft = oracle.transform_f64(img, method=0)
    F_dir = oracle.transform_f64(img, method=1)
    F_np = np.fft.fft2(img) / math.sqrt(img.size)
    assert np.max(np.abs(F_fft - F_dir)) < 1e-12
    assert np.max(np.abs(F_fft - F_np)) < 1e-12
    img = _rng(3).normal(0, 1, (256, 512))
    assert np.max(np.abs(oracle.transform_f64(img) - np.fft.fft2(img) / math.sqrt(img.size))) < 1e-11


def test_p1_delta_and_shift_sign(oracle):
    # a delta at (y0,x0) -> exp(-2 pi i (kx x0/W + ky y0/H))/sqrt(WH): pins the sign of the exponent
    H, W, y0, x0 = 16, 32, 3, 5
    img = np.zeros((H, W))
    img[y0, x0] = 1.0
    F = oracle.transform_f64(img)
    ky, kx = np.meshgrid(np.arange(H), np.arange(W), indexing="ij")
    expect = np.exp(-2j * np.pi * (kx * x0 / W + ky * y0 / H)) / math.sqrt(W * H)
    assert np.max(np.abs(F - expect)) < 1e-14


# ---- P2: Parseval pins the unitary scale (reading R1) -----------------------------------------
def test_p2_parseval(oracle):
    fr = _rng(4).integers(100, 4000, (6, 16, 32)).astype(np.uint16)
    lags = [1, 2, 4]
    r = oracle.structure_function(fr, lags, 8, want_2d=True)
    i_m = fr.astype(np.float64) / fr.reshape(6, -1).mean(axis=1)[:, None, None]
    for l, tau in enumerate(lags):
        real_space = np.mean([np.sum((i_m[t] - i_m[t + tau]) ** 2) for t in range(6 - tau)])
        assert abs(r.D2d[l].sum() - real_space) < 1e-12 * real_space
    assert abs(r.I2d.sum() - np.mean(np.sum(i_m ** 2, axis=(1, 2)))) < 1e-9


# ---- P3: normalisation --------------------------------------------------------------------------
def test_p3_constant_stack_gives_zero(oracle):
    one = _rng(5).integers(1, 60000, (32, 32)).astype(np.uint16)
    fr = np.repeat(one[None], 5, axis=0)
    r = oracle.structure_function(fr, [1, 2, 3], 8, want_2d=True)
    assert np.all(r.D2d == 0.0) and np.all(r.D == 0.0)
    assert r.I_q[1:].min() > 0


def test_p3_dc_is_zero_and_gain_invariance(oracle):
    base = _rng(6).integers(50, 500, (5, 16, 16)).astype(np.uint16)
    gains = np.array([1, 3, 7, 2, 5], dtype=np.uint16)
    r1 = oracle.structure_function(base, [1, 2], 6, want_2d=True)
    r2 = oracle.structure_function(base * gains[:, None, None], [1, 2], 6, want_2d=True)
    assert np.max(np.abs(r1.D2d[:, 0, 0])) < 1e-25           # F_t(0)=sqrt(WH) for every t
    assert abs(r1.I2d[0, 0] - 16 * 16) < 1e-10               # unitary scale: |F(0)|^2 = W H
    assert np.max(np.abs(r1.D2d - r2.D2d)) < 1e-12 * r1.D2d.max()
    assert np.max(np.abs(r1.D - r2.D)) < 1e-12 * r1.D.max()


def test_zero_mean_frame_is_an_error(oracle):
    fr = np.zeros((2, 8, 8), dtype=np.uint16)
    with pytest.raises(RuntimeError):
        oracle.structure_function(fr, [1], 4)


# ---- P4: travelling plane wave closed form (float input through the pure definition) -----------
def _plane_wave_frames(N, H, W, kx0, ky0, omega, A=1000.0, B=100.0):
    y, x = np.meshgrid(np.arange(H), np.arange(W), indexing="ij")
    return [A + B * np.cos(2 * np.pi * (kx0 * x / W + ky0 * y / H) - omega * t) for t in range(N)]


def test_p4_travelling_wave_closed_form(oracle):
    # D2d(+-k0,tau) = (B/2A)^2 WH (2 - 2 cos(omega tau)), zero elsewhere.  Uses the oracle's own
    # transform on float images (mean is exactly A), then the explicit pair loop in numpy here.
    N, H, W, kx0, ky0, om, A, B = 12, 16, 32, 5, 3, 0.37, 1000.0, 100.0
    F = [oracle.transform_f64(im / A) for im in _plane_wave_frames(N, H, W, kx0, ky0, om, A, B)]
    for tau in (1, 2, 5):
        D2d = np.mean([np.abs(F[t] - F[t + tau]) ** 2 for t in range(N - tau)], axis=0)
        expect = (B / (2 * A)) ** 2 * W * H * (2 - 2 * math.cos(om * tau))
        assert abs(D2d[ky0, kx0] - expect) < 1e-12 * expect
        assert abs(D2d[H - ky0, W - kx0] - expect) < 1e-12 * expect
        D2d[ky0, kx0] = D2d[H - ky0, W - kx0] = 0
        assert D2d.max() < 1e-20


def test_p4_p9_travelling_fringe_uint16_one_bin(oracle):
    # uint16 version through the whole oracle: D lands in exactly one |q| bin with value
    # 2 * closed form / c_b (plus the quantisation floor); pins pair loop + divisor + binning.
    N, H, W, kx0, ky0, om, A, B = 40, 32, 32, 6, 0, 0.5, 20000.0, 4000.0
    fr = np.array([np.rint(f) for f in _plane_wave_frames(N, H, W, kx0, ky0, om, A, B)]).astype(np.uint16)
    n_b = 16
    lags = [1, 3, 7]
    r = oracle.structure_function(fr, lags, n_b)
    b0 = int(math.floor(n_b * math.hypot(kx0 / W, ky0 / H) * 2))
    assert oracle.qbin(kx0, ky0, W, H, n_b) == b0
    for l, tau in enumerate(lags):
        expect = 2 * (B / (2 * A)) ** 2 * W * H * (2 - 2 * math.cos(om * tau)) / r.counts[b0]
        assert abs(r.D[l, b0] - expect) < 2e-4 * expect
        others = np.delete(r.D[l], b0)
        assert others.max() < 1e-4 * expect          # quantisation floor only
    assert r.n_pairs.tolist() == [N - 1, N - 3, N - 7]


def test_p9_static_fringe_one_I_bin_and_zero_D(oracle):
    N, H, W, kx0, ky0 = 4, 32, 64, 10, 4
    one = np.rint(_plane_wave_frames(1, H, W, kx0, ky0, 0.0, 20000.0, 4000.0)[0]).astype(np.uint16)
    fr = np.repeat(one[None], N, axis=0)
    n_b = 16
    r = oracle.structure_function(fr, [1, 2], n_b)
    assert np.all(r.D == 0)
    b0 = oracle.qbin(kx0, ky0, W, H, n_b)
    assert b0 == int(math.floor(n_b * 2 * math.hypot(kx0 / W, ky0 / H)))
    expect = 2 * (4000.0 / 40000.0) ** 2 * W * H / r.counts[b0]
    assert abs(r.I_q[b0] - expect) < 1e-3 * expect
    assert np.delete(r.I_q, b0).max() < 1e-5 * expect


# ---- P5: telegraph stack pins the lag indexing ------------------------------------------------------
def test_p5_telegraph(oracle):
    rng = _rng(7)
    P = rng.integers(100, 900, (16, 16)).astype(np.uint16)
    Q = rng.integers(100, 900, (16, 16)).astype(np.uint16)
    fr = np.array([P if t % 2 == 0 else Q for t in range(9)])
    lags = [1, 2, 3, 4, 5, 6]
    r = oracle.structure_function(fr, lags, 8, want_2d=True)
    dPQ = np.abs(oracle.transform_u16(P) - oracle.transform_u16(Q)) ** 2
    for l, tau in enumerate(lags):
        if tau % 2 == 0:
            assert np.all(r.D2d[l] == 0.0)
        else:
            assert np.max(np.abs(r.D2d[l] - dPQ)) < 1e-12 * dPQ.max()


# ---- P6: ramp pins the tau dependence ---------------------------------------------------------------
def test_p6_ramp(oracle):
    rng = _rng(8)
    I0 = rng.integers(2000, 3000, (16, 32)).astype(np.int64)
    G = rng.integers(-5, 6, (16, 32)).astype(np.int64)
    G.flat[0] -= G.sum()                                      # sum_x G = 0 -> mean constant
    N = 8
    fr = np.array([I0 + t * G for t in range(N)]).astype(np.uint16)
    lags = [1, 2, 3, 5]
    r = oracle.structure_function(fr, lags, 8, want_2d=True)
    FG2 = np.abs(np.fft.fft2(G / I0.mean()) / math.sqrt(G.size)) ** 2
    for l, tau in enumerate(lags):
        assert np.max(np.abs(r.D2d[l] - tau * tau * FG2)) < 1e-11 * FG2.max() * tau * tau


# ---- P7: linearity — the direct method A2 on tiny inputs --------------------------------
def test_p7_direct_method_equals_fourier_difference(oracle):
    fr = _rng(9).integers(10, 1000, (5, 8, 16)).astype(np.uint16)
    lags = [1, 2, 4]
    r = oracle.structure_function(fr, lags, 4, method=1, want_2d=True)
    i_m = fr.astype(np.float64) / fr.reshape(5, -1).mean(axis=1)[:, None, None]
    for l, tau in enumerate(lags):
        direct = np.mean([np.abs(oracle.transform_f64(i_m[t] - i_m[t + tau], method=1)) ** 2
                          for t in range(5 - tau)], axis=0)
        assert np.max(np.abs(direct - r.D2d[l])) < 1e-12 * direct.max()


# ---- P8: white noise: D = 2 sigma^2 = 2 I (north_star) -----------------------------------------------------
def test_p8_white_noise_flat(oracle):
    rng = _rng(10)
    N, H, W, mu, sig, n_b = 200, 32, 32, 10000.0, 300.0, 16
    fr = np.rint(rng.normal(mu, sig, (N, H, W))).astype(np.uint16)
    lags = [1, 5, 20]
    r = oracle.structure_function(fr, lags, n_b)
    var = (sig / mu) ** 2
    for b in range(n_b):
        if r.counts[b] == 0:
            continue
        tol = 6.0 / math.sqrt(r.counts[b] * (N - 20) / 2.0)
        assert abs(r.I_q[b] / var - 1.0) < tol
        for l in range(len(lags)):
            assert abs(r.D[l, b] / (2 * var) - 1.0) < tol
            assert abs(r.D[l, b] / (2 * r.I_q[b]) - 1.0) < tol


# ---- P9: binning + counts -----------------------------------------------------------------------------------
@pytest.mark.parametrize("W,H,n_b", [(64, 64, 32), (32, 64, 16), (128, 64, 50), (512, 512, 128)])
def test_p9_counts_bruteforce(oracle, W, H, n_b):
    r_counts = oracle.azimuthal_mean(np.ones((H, W)), n_b)[1]
    kx = np.arange(W)
    ky = np.arange(H)
    sx = np.where(kx < W // 2, kx, kx - W).astype(object)
    sy = np.where(ky < H // 2, ky, ky - H).astype(object)
    total = 0
    cnt = [0] * n_b
    for y in sy:
        for x in sx:
            if x == 0 and y == 0:
                continue
            num = 4 * (x * x * H * H + y * y * W * W)
            if num < W * W * H * H:
                total += 1
                cnt[math.isqrt(n_b * n_b * num // (W * W * H * H))] += 1
    assert int(r_counts.sum()) == total
    assert r_counts.tolist() == cnt
    if (W, H, n_b) == (64, 64, 32):
        assert total == 3204 and cnt[:8] == [0, 8, 16, 20, 24, 40, 36, 48]
    if (W, H, n_b) == (512, 512, 128):
        assert total == 205856 and cnt[:8] == [8, 36, 64, 84, 112, 132, 172, 184]


def test_p9_qbin_matches_python_ints_at_large_sizes(oracle):
    rng = _rng(11)
    for (W, H, n_b) in [(2048, 2048, 512), (4096, 4096, 1000), (4096, 32, 77)]:
        for _ in range(300):
            kx, ky = int(rng.integers(0, W)), int(rng.integers(0, H))
            assert oracle.qbin(kx, ky, W, H, n_b) == bf.qbin(kx, ky, W, H, n_b)


def test_p9_conservation(oracle):
    fr = _rng(12).integers(100, 4000, (5, 32, 32)).astype(np.uint16)
    n_b = 10
    r = oracle.structure_function(fr, [1, 2], n_b, want_2d=True)
    mask = np.array([[oracle.qbin(kx, ky, 32, 32, n_b) >= 0 for kx in range(32)] for ky in range(32)])
    for l in range(2):
        assert abs((r.counts * r.D[l]).sum() - r.D2d[l][mask].sum()) < 1e-12 * r.D2d[l].sum()
    assert abs((r.counts * r.I_q).sum() - r.I2d[mask].sum()) < 1e-12 * r.I2d[mask].sum()


# ---- P10: all-pairs identity ties D to I2d and the mean field ------------------------------------------------
def test_p10_all_pairs_identity(oracle):
    N = 7
    fr = _rng(13).integers(100, 4000, (N, 16, 16)).astype(np.uint16)
    lags = list(range(1, N))
    r = oracle.structure_function(fr, lags, 6, want_2d=True)
    F = np.array([oracle.transform_u16(f) for f in fr])
    lhs = sum((N - tau) * r.D2d[l] for l, tau in enumerate(lags))
    rhs = N * np.sum(np.abs(F) ** 2, axis=0) - np.abs(F.sum(axis=0)) ** 2
    assert np.max(np.abs(lhs - rhs)[1:, 1:]) < 1e-10 * rhs[1:, 1:].max()
    assert np.max(np.abs(r.I2d - np.mean(np.abs(F) ** 2, axis=0))[1:, 1:]) < 1e-12 * r.I2d[1:, 1:].max()


# ---- P12 / sampled variants equal the in-memory definition ---------------------------------------------------
def test_p12_windowed_and_sampled_equal_definition(oracle):
    fr = _rng(14).integers(100, 4000, (30, 32, 64)).astype(np.uint16)
    lags = [1, 2, 3, 5, 8, 13, 29, 30, 40]          # includes tau = N-1, tau = N and tau > N (R5)
    a = oracle.structure_function(fr, lags, 12, want_2d=True)
    w = oracle.structure_function(fr, lags, 12, want_2d=True, windowed=True)
    assert a.n_pairs.tolist() == [29, 28, 27, 25, 22, 17, 1, 0, 0] == w.n_pairs.tolist()
    assert np.all(a.D[7:] == 0) and np.all(w.D[7:] == 0)
    assert np.array_equal(a.counts, w.counts)
    assert np.max(np.abs(a.D2d - w.D2d)) < 1e-12 * a.D2d.max()
    assert np.max(np.abs(a.D - w.D)) < 1e-12 * a.D.max()
    assert np.max(np.abs(a.I_q - w.I_q)) < 1e-12 * a.I_q.max()
    ky = np.array([0, 1, 31, 16, 7])
    kx = np.array([1, 0, 63, 32, 50])
    s = oracle.structure_function_sampled(fr, lags, ky, kx)
    assert np.max(np.abs(s.D2d - a.D2d[:, ky, kx])) < 1e-12 * a.D2d.max()
    assert np.max(np.abs(s.I2d - a.I2d[ky, kx])) < 1e-12 * a.I2d.max()


# ---- P13: end-to-end golden vector ------------------------------------------------------------------------------
def _read_golden():
    g = {}
    for line in open(GOLDEN):
        if line.startswith("#") or not line.strip():
            continue
        k, *v = line.split()
        if k == "D":
            g.setdefault("D", {})[int(v[0])] = [float(x) for x in v[1:]]
        else:
            g[k] = [float(x) for x in v]
    return g


def test_p13_golden_vector(oracle):
    g = _read_golden()
    fr = np.array([[[100 + ((3 * x + 5 * y + 7 * t) % 11) for x in range(8)] for y in range(8)]
                   for t in range(4)]).astype(np.uint16)
    assert [oracle.frame_sum(f) for f in fr] == [int(s) for s in g["sums"]] == [6718, 6726, 6712, 6720]
    for method in (0, 1):
        r = oracle.structure_function(fr, [1, 2, 3], 4, method=method, want_2d=True)
        assert r.counts.tolist() == [int(c) for c in g["counts"]] == [0, 8, 16, 20]
        assert r.n_pairs.tolist() == [3, 2, 1]
        for l, tau in enumerate([1, 2, 3]):
            np.testing.assert_allclose(r.D[l], g["D"][tau], rtol=1e-11, atol=1e-20)
        np.testing.assert_allclose(r.I_q, g["I"], rtol=1e-11, atol=1e-20)
        assert abs(r.D2d[0, 0, 1] / g["D2d_ky0_kx1_tau1"][0] - 1) < 1e-11
        assert abs(r.D2d[0, 1, 0] / g["D2d_ky1_kx0_tau1"][0] - 1) < 1e-11
        assert abs(r.I2d[0, 0] - 64.0) < 1e-10 and r.D2d[0, 0, 0] < 1e-25
    # the survey's independently derived numbers, 12 digits
    survey_D1 = [0, 9.891985954380e-4, 1.043503054747e-3, 2.164191886320e-3]
    survey_I = [0, 2.680778101435e-4, 3.119287971524e-4, 9.509027718544e-4]
    np.testing.assert_allclose(g["D"][1], survey_D1, rtol=2e-12, atol=1e-20)
    np.testing.assert_allclose(g["I"], survey_I, rtol=2e-12, atol=1e-20)
    np.testing.assert_allclose(g["D"][2], [0, 2.216787015730e-4, 5.658843130045e-4, 2.315592755608e-3], rtol=2e-12)
    np.testing.assert_allclose(g["D"][3], [0, 8.178509086745e-4, 3.902731171114e-4, 1.481795127132e-3], rtol=2e-12)


# ---- P14: variance form of the fluctuation spectrum (oracle step 7) -------------------
def test_p14_variance_bruteforce_python_loops(oracle):
    # an independent statement in pure-Python loops (oracle/brute_force.py) on a tiny stack
    fr = _rng(21).integers(100, 4000, (5, 8, 8)).astype(np.uint16)
    r = oracle.variance_spectrum(fr, 4, want_2d=True)
    b = bf.variance_spectrum(fr.tolist(), 4)
    assert r.counts.tolist() == b["counts"]
    np.testing.assert_allclose(r.V2d, np.array(b["V2d"]), rtol=1e-10, atol=1e-18)
    np.testing.assert_allclose(r.V_q, np.array(b["V_q"]), rtol=1e-10)
    # method 1 (brute-force DFT inside the C oracle) agrees with the radix-2 path
    r1 = oracle.variance_spectrum(fr, 4, method=1, want_2d=True)
    np.testing.assert_allclose(r1.V2d, r.V2d, rtol=1e-9, atol=1e-18)


def test_p14_variance_is_tied_to_D_by_the_all_pairs_identity(oracle):
    # sum_tau (N - tau) D2d(k, tau) over ALL lags 1..N-1 = N^2 V2d(k): the pair loop (pinned by P4-P7, P10)
    # fixes the variance; a dropped mean, a 1/(N-1) divisor or a transposed map fails here
    N = 9
    fr = _rng(22).integers(100, 4000, (N, 16, 32)).astype(np.uint16)
    lags = list(range(1, N))
    d = oracle.structure_function(fr, lags, 8, want_2d=True)
    v = oracle.variance_spectrum(fr, 8, want_2d=True)
    lhs = sum((N - tau) * d.D2d[l] for l, tau in enumerate(lags)) / N ** 2
    assert np.max(np.abs(lhs - v.V2d)) < 1e-10 * v.V2d.max()
    assert np.array_equal(v.counts, d.counts)
    # binned: the same identity on the azimuthal means
    lhs_b = sum((N - tau) * d.D[l] for l, tau in enumerate(lags)) / N ** 2
    np.testing.assert_allclose(lhs_b, v.V_q, rtol=1e-10, atol=1e-18)


def test_p14_static_images_have_no_variance_and_gain_does_not_matter(oracle):
    one = np.rint(_plane_wave_frames(1, 32, 64, 10, 4, 0.0, 20000.0, 4000.0)[0]).astype(np.uint16)
    r = oracle.variance_spectrum(np.repeat(one[None], 6, axis=0), 16, want_2d=True)
    assert np.all(r.V2d < 1e-25) and np.all(r.V_q < 1e-25)     # a static fringe is in I(q), not in V(q)
    base = _rng(23).integers(50, 500, (5, 16, 16)).astype(np.uint16)
    gains = np.array([1, 3, 2, 7, 5], dtype=np.uint16)[:, None, None]
    a = oracle.variance_spectrum(base, 8, want_2d=True)
    b = oracle.variance_spectrum(base * gains, 8, want_2d=True)
    np.testing.assert_allclose(a.V2d, b.V2d, rtol=1e-9, atol=1e-22)


def test_p14_travelling_wave_closed_form(oracle):
    # I_t = A + B cos(k0.x - omega t) with omega N = 2 pi m: the field at +-k0 is (B/2A) sqrt(WH) e^{-+ i omega t},
    # its time mean vanishes over whole periods, so V2d(+-k0) = (B/2A)^2 WH exactly and 0 elsewhere
    N, H, W, kx0, ky0, A, B = 16, 16, 32, 5, 3, 1000.0, 100.0
    om = 2 * math.pi * 3 / N
    F = np.array([oracle.transform_f64(im / A) for im in _plane_wave_frames(N, H, W, kx0, ky0, om, A, B)])
    V = np.mean(np.abs(F - F.mean(axis=0)) ** 2, axis=0)
    expect = (B / (2 * A)) ** 2 * W * H
    assert abs(V[ky0, kx0] - expect) < 1e-12 * expect and abs(V[H - ky0, W - kx0] - expect) < 1e-12 * expect
    # and through the whole oracle on uint16 frames: one |q| bin holds 2 * expect / c_b (quantisation floor aside)
    A, B, n_b = 20000.0, 4000.0, 16
    fr = np.array([np.rint(f) for f in _plane_wave_frames(N, H, W, kx0, ky0, om, A, B)]).astype(np.uint16)
    r = oracle.variance_spectrum(fr, n_b)
    b0 = oracle.qbin(kx0, ky0, W, H, n_b)
    expect = 2 * (B / (2 * A)) ** 2 * W * H / r.counts[b0]
    assert abs(r.V_q[b0] - expect) < 2e-4 * expect
    assert np.delete(r.V_q, b0).max() < 1e-4 * expect


def test_p14_white_noise_variance_is_half_the_D_plateau(oracle):
    rng = _rng(24)
    N, H, W, mu, sig, n_b = 200, 32, 32, 10000.0, 300.0, 16
    fr = np.rint(rng.normal(mu, sig, (N, H, W))).astype(np.uint16)
    v = oracle.variance_spectrum(fr, n_b)
    var = (sig / mu) ** 2 * (1.0 - 1.0 / N)     # the sample mean takes 1/N of the variance
    for b in range(n_b):
        if v.counts[b]:
            assert abs(v.V_q[b] / var - 1.0) < 6.0 / math.sqrt(v.counts[b] * N / 2.0)


# ---- P11: the half-plane variant equals the full-plane definition --------------------------
def _synth_np(idx, **kw):
    import synth

    cfg = synth.config(idx, **kw)
    return cfg, synth.make_stack(cfg, "cpu").numpy()


@pytest.mark.parametrize("idx,kw", [(0, {}), (1, dict(W=128, N=60, lags=[1, 2, 3, 5, 8, 13, 21, 40], n_qbins=32)),
                                    (3, dict(W=64, N=24, lags=[1, 2, 7, 23, 24, 30], n_qbins=16))])
def test_p11_half_plane_equals_full_plane(oracle, idx, kw):
    """BASELINE.json configs[0] in full and scaled configs 1 and 3: the half-plane evaluation (Hermitian weights
    2 / 1 in the bin means) against the full-plane definition — counts identical, values to 1e-12."""
    cfg, fr = _synth_np(idx, **kw)
    full = oracle.structure_function(fr, cfg.lags, cfg.n_qbins, want_2d=True)
    half = oracle.structure_function_half(fr, cfg.lags, cfg.n_qbins, want_2d=True)
    assert np.array_equal(half.counts, full.counts) and np.array_equal(half.n_pairs, full.n_pairs)
    np.testing.assert_allclose(half.D, full.D, rtol=1e-12, atol=1e-300)
    np.testing.assert_allclose(half.I_q, full.I_q, rtol=1e-12, atol=1e-300)
    n = cfg.W // 2
    np.testing.assert_allclose(half.D2d, full.D2d[:, :, :n + 1], rtol=1e-12, atol=1e-22)
    np.testing.assert_allclose(half.I2d, full.I2d[:, :n + 1], rtol=1e-12, atol=1e-22)
    # rows with tau >= N are zero rows in both
    assert np.all(half.D[half.n_pairs == 0] == 0.0)


def test_p11_half_plane_counts_against_bruteforce_python_ints(oracle):
    """The weights 2 / 1 reproduce the full-plane counts of the pure-Python bin rule (oracle/brute_force.py), also on
    a non-square frame, where a transposed W/H in the weights or in the Nyquist column would show."""
    for (H, W, n_b) in ((8, 16, 5), (16, 8, 7), (32, 32, 16)):
        fr = _rng(31).integers(100, 4000, (3, H, W)).astype(np.uint16)
        half = oracle.structure_function_half(fr, [1, 2], n_b)
        c = [0] * n_b
        for ky in range(H):
            for kx in range(W):
                b = bf.qbin(kx, ky, W, H, n_b)
                if b >= 0:
                    c[b] += 1
        assert half.counts.tolist() == c
        full = oracle.structure_function(fr, [1, 2], n_b)
        np.testing.assert_allclose(half.D, full.D, rtol=1e-12, atol=1e-300)
