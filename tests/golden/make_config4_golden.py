"""Writes tests/golden/config4_golden.npz: the CPU oracle's values for BASELINE.json configs[4] at its full length
(1024^2 uint16 x 10 000 frames, lags 1..1000, 256 |q| bins), for ALL 1000 lags ("analyze all the time
delays"): the binned D of every lag, and the 2-D spectra of every lag on a sample of half-plane pixels.

Every stored value comes from oracle/ (nfs_oracle.structure_function_half: the plain fp64 definition of PAPER.md:L21,
L25, L31 on the half plane, pinned to the full-plane definition by P11); the input is the seeded synthetic stack of
synth.py (harness code, none of the method's arithmetic), generated on the GPU where one is present because the CPU
generator needs ~7 minutes for this stack.  Nothing of paper_1209_3362_b200 is imported.  The exact uint64 frame sums
of the stack are stored as a fingerprint: tests/test_gpu_full_size.py compares against this file only if its own stack
has the same fingerprint and recomputes the values through oracle_values() otherwise.

Run on a box with >= 128 GB of host memory (the oracle holds the half-plane transforms of all frames, 84 GB, and the
2-D sums of all lags, 4.2 GB); about half an hour on 16 cores (1.7e14 bytes of memory traffic):
    python tests/golden/make_config4_golden.py

Neither the lags nor the pixels are chosen with an eye on how the library tiles its work: all lags are stored, and the
pixels are the ones any checker of a half-plane spectrum would take (the neighbours of DC, both axes, the Nyquist
column and row) plus seeded random draws, half of them at low |q| where the signal of the synthetic stack lives.
If the stack on the testing box has other bytes (another generator device), the test falls back to a live oracle run on
FALLBACK_LAGS seeded random lags, which takes minutes instead of half an hour.
"""
import hashlib
import os
import sys

import numpy as np

ROOT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "..", "..")
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "config4_golden.npz")
FALLBACK_LAGS = 48


def fallback_lag_indices(n_lags):
    """Lag indices of the live fallback: the first, the last and FALLBACK_LAGS - 2 seeded random ones."""
    rng = np.random.default_rng(41)
    return sorted({0, n_lags - 1} | set(int(i) for i in rng.choice(np.arange(1, n_lags - 1), FALLBACK_LAGS - 2, replace=False)))


def sample_pixels(W, H):
    """Half-plane pixels (ky, kx): the neighbours of DC, both axes, the Nyquist column and row, then seeded random
    pixels: 24 at low |q| (where the signal of the synthetic stack lives) and 24 anywhere."""
    n = W // 2
    rng = np.random.default_rng(4)
    ky = [0, 1, 0, 1, H // 2, H - 1, 3, H // 4, 0, H // 2, 7]
    kx = [1, 0, 2, 1, 0, 1, n, n, n - 1, n, 0]
    ky += list(rng.integers(0, 24, 24)) + list(rng.integers(0, H, 24))
    kx += list(rng.integers(0, 24, 24)) + list(rng.integers(0, n + 1, 24))
    return np.array(ky, dtype=np.int64), np.array(kx, dtype=np.int64)


def fingerprint(frame_sums):
    return hashlib.sha256(np.ascontiguousarray(frame_sums, dtype=np.int64).tobytes()).hexdigest()


def oracle_values(host_stack, cfg, oracle, lag_idx=None):
    """host_stack: uint16 [N][H][W] numpy.  Returns the dict of arrays the test compares (oracle/ only): binned D, I,
    counts, pair counts and the sampled pixels of every 2-D spectrum, for the lags cfg.lags[lag_idx] (default: all)."""
    lag_idx = list(range(len(cfg.lags))) if lag_idx is None else list(lag_idx)
    lags = [cfg.lags[i] for i in lag_idx]
    ref = oracle.structure_function_half(host_stack, lags, cfg.n_qbins, want_2d=True)
    ky, kx = sample_pixels(cfg.W, cfg.H)
    return dict(D=ref.D, I_q=ref.I_q, counts=ref.counts, n_pairs=ref.n_pairs,
                D2d_pix=np.ascontiguousarray(ref.D2d[:, ky, kx]), I2d_pix=ref.I2d[ky, kx])


def main():
    import torch

    import synth
    from oracle import nfs_oracle

    cfg = synth.config(4)
    dev = "cuda" if torch.cuda.is_available() else "cpu"
    host = synth.make_stack(cfg, dev).cpu().numpy()   # the very call the test makes (same chunking of the generator)
    sums = host.reshape(cfg.N, -1).sum(axis=1, dtype=np.int64)
    vals = oracle_values(host, cfg, nfs_oracle)
    ky, kx = sample_pixels(cfg.W, cfg.H)
    np.savez_compressed(OUT, fingerprint=np.array(fingerprint(sums)), lag_idx=np.arange(len(cfg.lags)),
                        ky=ky, kx=kx, generated_on=np.array(dev), **vals)
    print("wrote", OUT, "fingerprint", fingerprint(sums), "device", dev, "lags", len(vals["n_pairs"]))


if __name__ == "__main__":
    main()
