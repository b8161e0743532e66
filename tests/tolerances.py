"""The numerical bars of the GPU parity tests, in one place ("Error model"; BASELINE.json north_star;
SURVEY.md §8(c) R15).

  TOL_BINNED   max relative error of the |q|-binned D(q,tau), I(q)
  TOL_PIXEL    max relative error of D2d(k,tau) wherever D2d > PIXEL_THRESHOLD * max D2d (max over the whole stored array)
  KAPPA        the absolute floor: below that threshold a relative bar means nothing and the error is bounded by
               KAPPA * max_k Z(k) E(k),  Z(k) = max_t |F_t(k) - F_0(k)|,  E(k) = max_t |F_t(k) - F_{t-1}(k)|
               — the size of one rounded term of the neighbouring-lag recurrence (an fp32 product of a reference-
               subtracted Fourier value and an increment), times a small chain factor.  DESIGN.md §6 derives it; the
               telegraph stack (exact zeros at even lags) measures 1.2 eps_fp32, a slowly drifting fringe 5 eps_fp32.

recurrence_floor() evaluates that bound from the ORACLE's spectra alone, through lower bounds of Z and E that hold for any
stack (so the tested bar is never looser than the stated one):
  |F_t - F_s| <= 2 Z  for all t, s            =>   Z(k) >= sqrt(max_tau D2d(k,tau)) / 2
  |F_t - F_{t-tau}| <= tau E                   =>   E(k) >= max_tau sqrt(D2d(k,tau)) / tau
"""
import numpy as np

TOL_BINNED = 1e-4
TOL_PIXEL = 1e-3
PIXEL_THRESHOLD = 1e-6
KAPPA = 1e-6


def recurrence_floor(D2d_ref, lags):
    """KAPPA * max_k Z_lb(k) E_lb(k) from oracle spectra D2d_ref [n_lags][...pixels...] at the given lags."""
    D = np.asarray(D2d_ref, dtype=np.float64)
    tau = np.asarray(lags, dtype=np.float64).reshape((-1,) + (1,) * (D.ndim - 1))
    Z_lb = 0.5 * np.sqrt(D.max(axis=0))
    E_lb = np.sqrt((D / tau ** 2).max(axis=0))
    return KAPPA * float((Z_lb * E_lb).max())
