"""Per-|q| fit of Eq. 1 (R19): D(b,tau) = A [1 - exp(-Gamma tau)] + C.
The oracle states R19's objective (the global least-squares minimiser over A, C, Gamma) and finds it by exhaustive
tabulation; it shares no search with the product.  Oracle pins (no GPU): exact recovery from noise-free model data,
invariances, agreement with scipy's least squares, no random (A, C, Gamma) with a smaller chi2, the flat far end of chi2.
GPU: nfs_fit_eq1 (whatever search it runs) must reach the oracle's objective value on the library's own binned D
and, where the minimum is sharp, its parameters; on a synthetic stack the fitted rate follows the generator's
Gamma(q) = gamma0 (q / q0)^2."""
import math

import numpy as np
import pytest

import synth
from oracle import fit_eq1 as ofit


def model(tau, A, C, G):
    return A * (1.0 - np.exp(-G * tau)) + C


@pytest.mark.parametrize("A,C,G", [(3.0, 0.2, 0.05), (1e-4, 3e-5, 0.8), (7.0, 0.0, 0.004), (2.0, 5.0, 2.5)])
def test_exact_recovery(A, C, G):
    tau = np.arange(1, 101, dtype=np.float64)
    a, c, g, chi2 = ofit.fit_bin(tau, model(tau, A, C, G))
    assert abs(g - G) / G < 1e-6 and abs(a - A) / A < 1e-6 and abs(c - C) <= 1e-6 * (A + C)
    assert chi2 < 1e-12 * (A + C) ** 2 * len(tau)


def test_invariances():
    rng = np.random.default_rng(3)
    tau = np.array(sorted(set(np.round(np.logspace(0, 2.7, 40)).astype(int))), dtype=np.float64)
    D = model(tau, 2.0, 0.3, 0.03) * (1.0 + 0.01 * rng.standard_normal(len(tau)))
    a, c, g, chi2 = ofit.fit_bin(tau, D)
    a2, c2, g2, chi22 = ofit.fit_bin(tau, 5.0 * D)                 # amplitude scale: A, C scale, Gamma stays
    assert np.allclose([a2, c2, g2, chi22], [5 * a, 5 * c, g, 25 * chi2], rtol=1e-6)
    a3, c3, g3, _ = ofit.fit_bin(tau, D + 1.5)                     # additive floor: only C moves
    assert np.allclose([a3, c3 - 1.5, g3], [a, c, g], rtol=1e-6, atol=1e-9)
    a4, c4, g4, _ = ofit.fit_bin(4.0 * tau, D)                     # time unit: Gamma scales inversely
    assert np.allclose([a4, c4, 4.0 * g4], [a, c, g], rtol=1e-6)
    assert ofit.fit_bin(tau[:2], D[:2]) == (0.0, 0.0, 0.0, 0.0)    # fewer than three lags


def test_against_scipy_least_squares():
    from scipy.optimize import least_squares

    rng = np.random.default_rng(11)
    tau = np.arange(1, 101, dtype=np.float64)
    for A, C, G in [(3.0, 0.2, 0.05), (1.0, 0.5, 0.3), (4.0, 0.1, 0.012)]:
        D = model(tau, A, C, G) + 0.02 * A * rng.standard_normal(len(tau))
        a, c, g, chi2 = ofit.fit_bin(tau, D)
        ref = least_squares(lambda p: model(tau, p[0], p[1], np.exp(p[2])) - D, x0=[a * 1.3, c * 0.5 + 0.01, np.log(g * 2.0)],
                            xtol=1e-15, ftol=1e-15, gtol=1e-15)
        assert np.allclose([a, c, g], [ref.x[0], ref.x[1], np.exp(ref.x[2])], rtol=2e-5)
        assert chi2 <= 2.0 * ref.cost * (1 + 1e-9) + 1e-18          # scipy's cost is half the sum of squares


def test_no_random_parameters_beat_the_oracle():
    """The defining property, probed directly on the objective written out (chi2_of): nothing drawn from the allowed
    box, nor from a tight cloud around the answer, has a smaller sum of squared residuals."""
    rng = np.random.default_rng(5)
    tau = np.array([1, 2, 3, 4, 6, 8, 11, 16, 23, 32, 45, 64, 91, 128], dtype=np.float64)
    D = model(tau, 2.0, 0.4, 0.07) * (1.0 + 0.05 * rng.standard_normal(len(tau)))
    a, c, g, chi2 = ofit.fit_bin(tau, D)
    assert abs(ofit.chi2_of(a, c, g, tau, D) - chi2) <= 1e-12 * chi2
    lo, hi = 1e-3 / tau.max(), 1e2 / tau.min()
    for _ in range(4000):
        G = math.exp(rng.uniform(math.log(lo), math.log(hi)))
        assert ofit.chi2_of(rng.uniform(-1, 5), rng.uniform(-1, 3), G, tau, D) >= chi2
    for _ in range(4000):
        da, dc, dg = 1e-3 * rng.standard_normal(3)
        assert ofit.chi2_of(a * (1 + da), c * (1 + dc), g * (1 + dg), tau, D) >= chi2 * (1 - 1e-12)


def test_far_plateau_of_chi2_is_not_returned():
    """Two relaxation processes far apart: chi2_min(Gamma) has its valley at the slow rate and, at rates so high that
    1 - exp(-Gamma tau) = 1 for every lag, a flat shelf with a shallow dip.  A local search started on the shelf stays
    there; the oracle must return the valley, which the same local search finds when started beside it."""
    from scipy.optimize import least_squares

    tau = np.array(sorted(set(np.round(np.logspace(0, 3, 40)).astype(int))), dtype=np.float64)
    D = (1.0 - np.exp(-1.0 * tau)) + (1.0 - np.exp(-0.003 * tau))
    a, c, g, chi2 = ofit.fit_bin(tau, D)
    res = lambda p: model(tau, p[0], p[1], np.exp(p[2])) - D
    shelf = least_squares(res, x0=[0.1, 1.8, np.log(26.0)], xtol=1e-15, ftol=1e-15, gtol=1e-15)
    valley = least_squares(res, x0=[1.0, 1.0, np.log(0.005)], xtol=1e-15, ftol=1e-15, gtol=1e-15)
    assert np.exp(shelf.x[2]) > 5.0 and 2.0 * shelf.cost > 10.0 * chi2
    assert np.allclose([a, c, g], [valley.x[0], valley.x[1], np.exp(valley.x[2])], rtol=2e-5)
    assert abs(chi2 - 2.0 * valley.cost) <= 1e-6 * chi2


def test_fit_all_bins_skips_empty_bins_and_lags_without_pairs():
    tau = [1, 2, 3, 5, 8, 13, 21, 400]
    D = np.stack([model(np.array(tau, float), 1.0 + b, 0.1, 0.1 * (b + 1)) for b in range(3)], axis=1)
    n_pairs = np.array([99, 98, 97, 95, 92, 87, 79, 0])
    D[-1] = 0.0
    A, C, G, chi2 = ofit.fit_eq1(tau, n_pairs, np.array([4, 0, 8]), D)
    assert A[1] == C[1] == G[1] == chi2[1] == 0.0
    assert np.allclose(A[[0, 2]], [1.0, 3.0], rtol=1e-6) and np.allclose(G[[0, 2]], [0.1, 0.3], rtol=1e-6)


@pytest.mark.gpu
def test_gpu_fit_matches_oracle_and_generator():
    import torch

    from paper_1209_3362_b200 import binding

    assert torch.cuda.is_available()
    lags = list(range(1, 41)) + [50, 64, 80, 100, 128, 160, 600]
    cfg = synth.config(1, W=128, N=500, lags=lags, n_qbins=32)
    st = synth.make_stack(cfg, "cuda")
    nfs = binding.NFS(cfg.W, cfg.H, lags, cfg.n_qbins)
    nfs.push(st)
    D, I_q, cnt = nfs.finalize()
    npairs = nfs.pair_counts()
    A, C, G, chi2 = nfs.fit_eq1()
    V = nfs.variance()
    nfs.close()
    assert npairs[-1] == 0                                          # lag 600 >= N: left out of the fit
    oA, oC, oG, ochi2 = ofit.fit_eq1(lags, npairs, cnt, D)          # the oracle (global minimiser) on the same binned D
    nz = cnt > 0
    assert np.all(A[~nz] == 0) and np.all(G[~nz] == 0)
    # (1) the objective: the library's chi2 is what its own (A, C, Gamma) give when put into the objective written out
    tt = np.array(lags[:-1], dtype=np.float64)
    for b in np.flatnonzero(nz):
        own = ofit.chi2_of(A[b], C[b], G[b], tt, D[:-1, b])
        assert abs(own - chi2[b]) <= 1e-9 * own + 1e-30, (b, own, chi2[b])
    # (2) ... and it is the global minimum: not above the oracle's by more than 1e-6 relative in any bin (nor below it
    # by more: that would mean the oracle missed the minimum)
    floor = 1e-16 * np.abs(oA).max() ** 2
    assert np.all(chi2[nz] <= ochi2[nz] * (1 + 1e-6) + floor), np.max(chi2[nz] / ochi2[nz])
    assert np.all(ochi2[nz] <= chi2[nz] * (1 + 1e-6) + floor), np.max(ochi2[nz] / chi2[nz])
    # (3) the parameters, at 1e-4, where the minimum is sharp (signal well above the noise floor); in noise-dominated
    # bins chi2 is flat in Gamma (A ~ 0 leaves Gamma undetermined) and only (1), (2) are meaningful
    sharp = nz & (oA > 20 * np.abs(oC))
    assert sharp.sum() >= 5
    assert np.allclose(G[sharp], oG[sharp], rtol=1e-4)
    assert np.allclose(A[sharp], oA[sharp], rtol=1e-4)
    assert np.allclose(C[sharp], oC[sharp], rtol=1e-4, atol=1e-5 * np.abs(oA[sharp]).min())
    # physics of the synthetic stack (generator statistics, loose): where the signal dominates the fitted rate grows
    # like q^2 and the plateau A + C approaches twice the variance form (Eq. 1 with f -> 0)
    q = (np.arange(cfg.n_qbins) + 0.5) / cfg.n_qbins * 0.5          # cycles per pixel at the bin centres
    sel = nz & (A > 20 * np.abs(C)) & (G * max(lags[:-1]) > 3) & (G < 0.5)
    assert sel.sum() >= 3
    slope = np.polyfit(np.log(q[sel]), np.log(G[sel]), 1)[0]
    assert 1.5 < slope < 2.5
    assert np.allclose((A + C)[sel], 2 * V[sel], rtol=0.15)
