"""Writes tests/golden/config4_golden.npz: the CPU oracle's values for BASELINE.json configs[4] at its full length
(1024^2 uint16 x 10 000 frames, lags 1..1000, 256 |q| bins), for 55 of the 1000 lags.

Every stored value comes from oracle/ (nfs_oracle.structure_function_half: the plain fp64 definition of PAPER.md:L21,
L25, L31 on the half plane, pinned to the full-plane definition by P11); the input is the seeded synthetic stack of
synth.py (harness code, none of the method's arithmetic), generated on the GPU where one is present because the CPU
generator needs ~7 minutes for this stack.  Nothing of paper_1209_3362_b200 is imported.  The exact uint64 frame sums
of the stack are stored as a fingerprint: tests/test_gpu_full_size.py compares against this file only if its own stack
has the same fingerprint and recomputes the values through oracle_values() otherwise.

Run on a box with >= 128 GB of host memory (the oracle holds the half-plane transforms of all frames: 84 GB):
    python tests/golden/make_config4_golden.py
"""
import hashlib
import os
import sys

import numpy as np

ROOT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "..", "..")
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "config4_golden.npz")
# lags (as indices into the lag list) whose 2-D spectra are compared on the sampled pixels
PIXEL_LAG_INDICES = [0, 12, 13, 103, 104, 500, 998, 999]


def selected_lag_indices(n_lags):
    """55 of the 1000 lag indices (at most 64): the short lags, a log-spaced ladder, both sides of every boundary between the lag groups
    and lag tasks the library is likely to form (multiples of 13 and 104), and the longest lags."""
    sel = set(range(0, 8)) | set(PIXEL_LAG_INDICES) | {n_lags - 1, n_lags - 2, n_lags - 14}
    for k in range(1, 10):
        sel |= {104 * k - 1, 104 * k}
    v = 10.0
    while v < n_lags:
        sel.add(int(v))
        v *= 1.22
    sel = sorted(i for i in sel if 0 <= i < n_lags)
    step = max(1, len(sel) // 64)
    keep = set(PIXEL_LAG_INDICES) | {n_lags - 1}
    out = [i for k, i in enumerate(sel) if i in keep or k % step == 0]
    return out[:64] if len(out) > 64 else out


def sample_pixels(W, H):
    """Half-plane pixels (ky, kx): next to DC, the axes, the Nyquist column, the low-|q| region where the signal lives,
    and uniform samples."""
    n = W // 2
    rng = np.random.default_rng(4)
    ky = [0, 1, 0, 1, H // 2, H - 1, 3, H // 4, 0, H // 2, 7]
    kx = [1, 0, 2, 1, 0, 1, n, n, n - 1, n, 0]
    ky += list(rng.integers(0, 24, 24)) + list(rng.integers(0, H, 24))
    kx += list(rng.integers(0, 24, 24)) + list(rng.integers(0, n + 1, 24))
    return np.array(ky, dtype=np.int64), np.array(kx, dtype=np.int64)


def fingerprint(frame_sums):
    return hashlib.sha256(np.ascontiguousarray(frame_sums, dtype=np.int64).tobytes()).hexdigest()


def oracle_values(host_stack, cfg, oracle):
    """host_stack: uint16 [N][H][W] numpy.  Returns the dict of arrays the test compares (oracle/ only)."""
    lag_idx = selected_lag_indices(len(cfg.lags))
    lags = [cfg.lags[i] for i in lag_idx]
    ref = oracle.structure_function_half(host_stack, lags, cfg.n_qbins, want_2d=True)
    ky, kx = sample_pixels(cfg.W, cfg.H)
    rows = [lag_idx.index(l) for l in PIXEL_LAG_INDICES]
    return dict(D=ref.D, I_q=ref.I_q, counts=ref.counts, n_pairs=ref.n_pairs,
                D2d_pix=np.stack([ref.D2d[r][ky, kx] for r in rows]), I2d_pix=ref.I2d[ky, kx])


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
    np.savez_compressed(OUT, fingerprint=np.array(fingerprint(sums)), lag_idx=np.array(selected_lag_indices(len(cfg.lags))),
                        ky=ky, kx=kx, generated_on=np.array(dev), **vals)
    print("wrote", OUT, "fingerprint", fingerprint(sums), "device", dev, "lags", len(vals["n_pairs"]))


if __name__ == "__main__":
    main()
