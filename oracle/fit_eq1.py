"""oracle/fit_eq1.py — CPU ORACLE (test infrastructure, not the product) of the per-|q| fit of Eq. 1.

PAPER.md:L23-25, Eq. 1:  <|Delta I_m(q,tau)|^2> = 2a { T(q) I_s(q) [1 - f(q,tau)] + B(q) }.  With the azimuthally averaged
structure function D(b,tau) of |q| bin b this reads  D(b,tau) = A_b [1 - f_b(tau)] + C_b,  A_b = 2a T I_s (the signal
plateau) and C_b = 2a B (the noise floor).  The paper obtains I_s and f "by analyzing the time delay dependence" and
does not print a procedure; the reading adopted here (R19) is the usual one for diffusive concentration
fluctuations (refs. 4, 5 of the paper): f_b(tau) = exp(-Gamma_b tau), and the fit is DEFINED by its objective:

    (A, C, Gamma)  =  the global minimiser of   chi2(A, C, Gamma) = sum_l [ D_l - A (1 - exp(-Gamma tau_l)) - C ]^2
                      over all real A, C and all Gamma in [1e-3 / tau_max, 1e2 / tau_min],

the sum running over the lags that have at least one frame pair (unweighted least squares).  Fewer than three usable
lags, or an empty |q| bin: all four outputs are 0.

This file states that objective and finds its minimiser by exhaustion, not by any clever search, so that a reader can
check it against the definition by eye and so that it shares nothing with whatever search the product uses:

  * for ONE trial Gamma the model is linear in (A, C): the best pair is the least-squares solution of the L x 2 system
    [1 - exp(-Gamma tau_l), 1] (A, C)^T ~ D_l, obtained from the library routine numpy.linalg.lstsq;  chi2_min(Gamma)
    is the squared residual of that solution;
  * chi2_min is tabulated on N_GRID = 20001 log-equidistant rates covering the whole interval; the smallest entry (the
    first one, if several tie) locates the global minimum to one grid step (1e-3 in log Gamma for typical lag lists —
    far finer than any structure chi2_min can have for at most a few hundred lags);
  * the two grid cells around it are tabulated again with N_ZOOM = 2001 points, and so on, until the step in
    log Gamma is below 1e-13: the grid point of smallest chi2_min is the answer.

Pins (tests/test_fit_eq1.py): exact recovery of (A, C, Gamma) from noise-free model data; scale / offset / time-unit
invariances; agreement with scipy.optimize.least_squares started near the answer; no randomly drawn (A, C, Gamma)
anywhere in the allowed box has a smaller chi2; a case where a local search started on the flat far end of chi2 is
beaten.  Plain numpy, fp64.
"""
import math

import numpy as np

N_GRID = 20001
N_ZOOM = 2001
MIN_STEP = 1e-13


def chi2_of(A, C, Gamma, tau, D):
    """The objective itself, written out: sum_l [D_l - A (1 - exp(-Gamma tau_l)) - C]^2."""
    r = D - A * (1.0 - np.exp(-Gamma * tau)) - C
    return float(np.dot(r, r))


def best_A_C(Gamma, tau, D):
    """For a fixed rate the model is linear in (A, C): their least-squares values from numpy.linalg.lstsq, and the
    squared residual they leave."""
    M = np.column_stack([-np.expm1(-Gamma * tau), np.ones_like(tau)])  # 1 - exp(-Gamma tau), evaluated without cancellation
    (A, C), _, _, _ = np.linalg.lstsq(M, D, rcond=None)
    r = D - M @ np.array([A, C])
    return float(A), float(C), float(np.dot(r, r))


def _tabulate(xs, tau, D):
    return np.array([best_A_C(math.exp(x), tau, D)[2] for x in xs])


def fit_bin(tau, D):
    """One |q| bin: tau [L] > 0, D [L].  Returns (A, C, Gamma, chi2) of the global minimum."""
    tau = np.asarray(tau, dtype=np.float64)
    D = np.asarray(D, dtype=np.float64)
    if len(tau) < 3:
        return 0.0, 0.0, 0.0, 0.0
    lo = math.log(1e-3 / tau.max())
    hi = math.log(1e2 / tau.min())
    xs = np.linspace(lo, hi, N_GRID)
    while True:
        chis = _tabulate(xs, tau, D)
        k = int(np.argmin(chis))  # first smallest
        step = xs[1] - xs[0]
        if step < MIN_STEP:
            break
        xs = np.linspace(xs[max(k - 1, 0)], xs[min(k + 1, len(xs) - 1)], N_ZOOM)
    x = float(xs[k])
    A, C, chi2 = best_A_C(math.exp(x), tau, D)
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
