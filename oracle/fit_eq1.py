"""oracle/fit_eq1.py — CPU ORACLE (test infrastructure, not the product) of the per-|q| fit of Eq. 1.

PAPER.md:L23-25, Eq. 1:  <|Delta I_m(q,tau)|^2> = 2a { T(q) I_s(q) [1 - f(q,tau)] + B(q) }.  With the azimuthally averaged
structure function D(b,tau) of |q| bin b this reads  D(b,tau) = A_b [1 - f_b(tau)] + C_b,  A_b = 2a T I_s (the signal
plateau) and C_b = 2a B (the noise floor).  The paper obtains I_s and f "by analyzing the time delay dependence" and
does not print the procedure; the reading adopted here (R19) is the usual one for diffusive concentration
fluctuations (refs. 4, 5 of the paper): f_b(tau) = exp(-Gamma_b tau), fitted by unweighted least squares over the lags
that have at least one frame pair.  Because this is an iteration, the oracle follows the algorithm step by step:

  1. x = log Gamma is searched on [log(1e-3 / tau_max), log(1e2 / tau_min)];
  2. for a trial x:  g_l = 1 - exp(-Gamma tau_l);  (A, C) = the linear least-squares solution of D_l ~ A g_l + C
     (2 x 2 normal equations; A = 0, C = mean D if they are singular);  chi2(x) = sum_l (D_l - A g_l - C)^2;
  3. chi2 on a grid of 64 equidistant x; k* = the first grid point of smallest chi2;
  4. golden-section search, 48 iterations, on [x_{k*-1}, x_{k*+1}] (clipped to the grid);
  5. Gamma = exp of the final interval's midpoint, (A, C, chi2) evaluated there.
Fewer than three usable lags, or an empty |q| bin: all four outputs are 0.

Pins (tests/test_fit_eq1.py): exact recovery of (A, C, Gamma) from noise-free model data, scale / offset / time-unit
invariances, and agreement with scipy.optimize.least_squares on noisy data.  Plain numpy, fp64.
"""
import math

import numpy as np

GRID = 64
GOLDEN_ITERS = 48
INV_PHI = (math.sqrt(5.0) - 1.0) / 2.0


def _linear(x, tau, D):
    """Step 2: (A, C, chi2) at log-rate x."""
    g = -np.expm1(-math.exp(x) * tau)
    n = float(len(tau))
    Sg, Sgg, Sd, Sgd = g.sum(), (g * g).sum(), D.sum(), (g * D).sum()
    det = n * Sgg - Sg * Sg
    if det <= 1e-14 * n * Sgg:
        A, C = 0.0, Sd / n
    else:
        A = (n * Sgd - Sg * Sd) / det
        C = (Sd - A * Sg) / n
    r = D - A * g - C
    return A, C, float((r * r).sum())


def fit_bin(tau, D):
    """One |q| bin: tau [L] > 0, D [L].  Returns (A, C, Gamma, chi2)."""
    tau = np.asarray(tau, dtype=np.float64)
    D = np.asarray(D, dtype=np.float64)
    if len(tau) < 3:
        return 0.0, 0.0, 0.0, 0.0
    lo = math.log(1e-3 / tau.max())
    hi = math.log(1e2 / tau.min())
    xs = [lo + (hi - lo) * k / (GRID - 1) for k in range(GRID)]
    chis = [_linear(x, tau, D)[2] for x in xs]
    k = int(np.argmin(chis))          # first smallest
    a, c = xs[max(k - 1, 0)], xs[min(k + 1, GRID - 1)]
    x1 = c - INV_PHI * (c - a)
    x2 = a + INV_PHI * (c - a)
    f1, f2 = _linear(x1, tau, D)[2], _linear(x2, tau, D)[2]
    for _ in range(GOLDEN_ITERS):
        if f1 <= f2:
            c, x2, f2 = x2, x1, f1
            x1 = c - INV_PHI * (c - a)
            f1 = _linear(x1, tau, D)[2]
        else:
            a, x1, f1 = x1, x2, f2
            x2 = a + INV_PHI * (c - a)
            f2 = _linear(x2, tau, D)[2]
    x = 0.5 * (a + c)
    A, C, chi2 = _linear(x, tau, D)
    return A, C, math.exp(x), chi2


def fit_eq1(lags, n_pairs, counts, D):
    """All bins: lags [n_l], n_pairs [n_l] (lags without a pair are left out), counts [n_b] (empty bins give zeros),
    D [n_l][n_b].  Returns A, C, Gamma, chi2, each [n_b]."""
    lags = np.asarray(lags, dtype=np.float64)
    use = np.asarray(n_pairs) > 0
    nb = D.shape[1]
    out = np.zeros((4, nb))
    for b in range(nb):
        if counts[b] > 0:
            out[:, b] = fit_bin(lags[use], D[use, b])
    return out[0], out[1], out[2], out[3]
