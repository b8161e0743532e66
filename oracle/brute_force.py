"""oracle/brute_force.py — the definition in pure-Python loops (tiny inputs only).

CPU ORACLE, TEST INFRASTRUCTURE, NOT THE PRODUCT.  Second, independent statement of SURVEY.md
§8(c) steps 1-6 (PAPER.md:L21 normalise by the spatial mean; L25 spatial Fourier transform,
power spectrum, average over the measurement time, azimuthal average; L31 N-tau pairs per lag),
written with explicit loops, Python ints and cmath only — no numpy, no FFT, no C.  It exists so
that oracle/nfs_oracle.c can be pinned against something that is not itself, and it writes the
golden vector tests/golden/p13_golden.txt (via tests/golden/make_p13_golden.py).
Cost is O(N (WH)^2): keep W,H <= 16.
"""
import cmath
import math


def normalise(frame):
    """frame: list of H rows of W ints -> (S_t, rows of floats I/m_t)   [step 1, L21]"""
    H, W = len(frame), len(frame[0])
    S = 0
    for row in frame:
        for v in row:
            S += int(v)
    if S == 0:
        raise ZeroDivisionError("frame sums to zero")
    m = S / (W * H)
    return S, [[int(v) / m for v in row] for row in frame]


def dft2_unitary(img):
    """F(ky,kx) = (1/sqrt(WH)) sum_{y,x} img[y][x] exp(-2 pi i (kx x/W + ky y/H))   [step 2]"""
    H, W = len(img), len(img[0])
    scale = 1.0 / math.sqrt(W * H)
    F = [[0j] * W for _ in range(H)]
    for ky in range(H):
        for kx in range(W):
            s = 0j
            for y in range(H):
                for x in range(W):
                    # exact rational phase: ((kx x mod W) H + (ky y mod H) W) / (W H)
                    num = ((kx * x) % W) * H + ((ky * y) % H) * W
                    s += img[y][x] * cmath.exp(-2j * math.pi * (num % (W * H)) / (W * H))
            F[ky][kx] = s * scale
    return F


def qbin(kx, ky, W, H, n_b):
    """step 5: exact-integer |q| bin of full-plane FFT-order pixel; -1 if excluded"""
    sx = kx if kx < W // 2 else kx - W
    sy = ky if ky < H // 2 else ky - H
    if sx == 0 and sy == 0:
        return -1
    q = (4 * n_b * n_b * (sx * sx * H * H + sy * sy * W * W)) // (W * W * H * H)
    b = math.isqrt(q)
    return b if b < n_b else -1


def structure_function(frames, lags, n_b):
    """frames: list of N frames (list of rows of ints).  Returns dict with
    sums, D2d[l][ky][kx], I2d[ky][kx], D[l][b], I_q[b], counts[b], n_pairs[l]."""
    N = len(frames)
    H, W = len(frames[0]), len(frames[0][0])
    sums, F = [], []
    for fr in frames:
        S, im = normalise(fr)
        sums.append(S)
        F.append(dft2_unitary(im))
    D2d, n_pairs = [], []
    for tau in lags:
        acc = [[0.0] * W for _ in range(H)]
        npair = N - tau if tau < N else 0
        for t in range(npair):                                   # step 3: explicit pair loop
            for ky in range(H):
                for kx in range(W):
                    d = F[t][ky][kx] - F[t + tau][ky][kx]
                    acc[ky][kx] += d.real * d.real + d.imag * d.imag
        if npair:
            acc = [[v / npair for v in row] for row in acc]
        D2d.append(acc)
        n_pairs.append(npair)
    I2d = [[sum(abs(F[t][ky][kx]) ** 2 for t in range(N)) / N for kx in range(W)] for ky in range(H)]  # step 4

    def azimuthal(m2d):                                          # steps 5-6
        s = [0.0] * n_b
        c = [0] * n_b
        for ky in range(H):
            for kx in range(W):
                b = qbin(kx, ky, W, H, n_b)
                if b >= 0:
                    s[b] += m2d[ky][kx]
                    c[b] += 1
        return [s[b] / c[b] if c[b] else 0.0 for b in range(n_b)], c

    D = [azimuthal(m)[0] for m in D2d]
    I_q, counts = azimuthal(I2d)
    return dict(sums=sums, D2d=D2d, I2d=I2d, D=D, I_q=I_q, counts=counts, n_pairs=n_pairs)


def variance_spectrum(frames, n_b):
    """Step 7: V2d = (1/N) sum_t |F_t - <F>_t|^2 per pixel and its azimuthal mean,
    in explicit loops.  Returns dict with V2d[ky][kx], V_q[b], counts[b]."""
    N = len(frames)
    H, W = len(frames[0]), len(frames[0][0])
    F = [dft2_unitary(normalise(fr)[1]) for fr in frames]
    V2d = [[0.0] * W for _ in range(H)]
    for ky in range(H):
        for kx in range(W):
            m = sum(F[t][ky][kx] for t in range(N)) / N
            V2d[ky][kx] = sum(abs(F[t][ky][kx] - m) ** 2 for t in range(N)) / N
    s = [0.0] * n_b
    c = [0] * n_b
    for ky in range(H):
        for kx in range(W):
            b = qbin(kx, ky, W, H, n_b)
            if b >= 0:
                s[b] += V2d[ky][kx]
                c[b] += 1
    return dict(V2d=V2d, V_q=[s[b] / c[b] if c[b] else 0.0 for b in range(n_b)], counts=c)
