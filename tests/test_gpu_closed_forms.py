"""The CUDA path against what the mathematics fixes directly (the same closed forms that pin the oracle, SURVEY.md
§8(c) P3-P6, P9) and the variance form of the fluctuation spectrum against oracle step 7.  The full-size comparisons
with the oracle are in tests/test_gpu_full_size.py."""
import numpy as np
import pytest
import torch

import synth
from tolerances import KAPPA, TOL_PIXEL, recurrence_floor

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def binding():
    assert torch.cuda.is_available()
    from paper_1209_3362_b200 import binding as b

    b.load_library()
    return b


def run(binding, stack_np, lags, n_b, batch=0, direct=False):
    st = torch.from_numpy(np.ascontiguousarray(stack_np)).cuda()
    N, H, W = st.shape
    nfs = binding.NFS(W, H, lags, n_b, batch_frames=batch, direct=direct)
    nfs.push(st)
    D, I_q, cnt = nfs.finalize()
    D2d = np.stack([nfs.D2d(l) for l in range(len(lags))])
    I2d = nfs.I2d()
    nfs.close()
    return D, I_q, cnt, D2d, I2d


def test_constant_stack_gives_exact_zero(binding):
    """P3: identical frames => every difference vanishes (L21); with the reference subtraction exactly."""
    rng = np.random.default_rng(5)
    img = rng.integers(100, 4000, size=(64, 64)).astype(np.uint16)
    D, I_q, cnt, D2d, I2d = run(binding, np.repeat(img[None], 12, 0), [1, 2, 3, 7], 16)
    assert np.all(D == 0.0) and np.all(D2d == 0.0)
    assert I2d[0, 0] == pytest.approx(64 * 64, rel=1e-6)       # unitary scale: |F(0)|^2 = W H (reading R1)


def test_gain_invariance(binding):
    """P3: multiplying frame t by an integer gain leaves every output unchanged (normalisation by the mean, L21)."""
    cfg = synth.config(0)
    st = synth.make_stack(cfg, "cpu", n=12).numpy().astype(np.int64)
    gains = np.array([1, 2, 3, 1, 5, 2, 1, 4, 3, 2, 1, 6])[:, None, None]
    a = run(binding, st.astype(np.uint16), [1, 2, 3], 16)
    b = run(binding, (st * gains).astype(np.uint16), [1, 2, 3], 16)
    nz = a[2] > 0
    assert np.abs(a[0][:, nz] - b[0][:, nz]).max() / a[0][:, nz].max() < 1e-5
    assert np.abs(a[1][nz] - b[1][nz]).max() / a[1][nz].max() < 1e-5


def test_telegraph_stack(binding):
    """P5: frames alternate between P and Q: even lags give 0, odd lags |F_P - F_Q|^2 for every tau.  Lags that open a
    run of consecutive lags (or stand alone) are accumulated directly and give exact zeros; the further lags of a run
    come from the neighbouring-lag recurrence and give zero up to the absolute floor of DESIGN.md §6
    (tests/tolerances.py: here Z = E = |F_P - F_Q|, so the floor is KAPPA / 2 times the odd-lag value)."""
    rng = np.random.default_rng(7)
    Pimg = rng.integers(500, 3000, size=(64, 64)).astype(np.uint16)
    Qimg = rng.integers(500, 3000, size=(64, 64)).astype(np.uint16)
    st = np.stack([Pimg if t % 2 == 0 else Qimg for t in range(21)])
    lags = [1, 2, 3, 4, 5, 6, 9, 12]
    D, I_q, cnt, D2d, I2d = run(binding, st, lags, 16, batch=8)
    ip = Pimg / Pimg.mean()
    iq = Qimg / Qimg.mean()
    ref = np.abs(np.fft.rfft2(ip - iq, norm="ortho")) ** 2
    floor = recurrence_floor(np.stack([ref * (tau % 2) for tau in lags]), lags)
    assert floor == pytest.approx(0.5 * KAPPA * ref.max(), rel=1e-12)
    for l, tau in enumerate(lags):
        if tau % 2 == 0:
            assert np.abs(D2d[l]).max() <= floor
            if tau == 12:
                assert np.all(D2d[l] == 0.0)
        else:
            m = ref > 1e-6 * ref.max()
            assert (np.abs(D2d[l] - ref)[m] / ref[m]).max() < 1e-4
    # NFS_FLAG_DIRECT: no recurrence anywhere, so every even lag is an exact zero again
    Dd, _, _, D2d_direct, _ = run(binding, st, lags, 16, batch=8, direct=True)
    for l, tau in enumerate(lags):
        if tau % 2 == 0:
            assert np.all(D2d_direct[l] == 0.0) and np.all(Dd[l] == 0.0)
        else:
            m = ref > 1e-6 * ref.max()
            assert (np.abs(D2d_direct[l] - ref)[m] / ref[m]).max() < 1e-4


def test_slowly_drifting_fringe_keeps_small_lags_accurate(binding):
    """The accuracy contract of include/nfs.h (DESIGN.md §6 error model).  A fringe that creeps by 0.0005 rad
    per frame for 1200 frames: at its pixel the excursion from the reference frame, Z = max |F_t - F_0|, is 1100 times the
    frame-to-frame increment E, and D(tau = 1) is less than a millionth of Z^2.  Lags inside a run come from the
    neighbouring-lag recurrence, whose rounding error scales with Z E and not with D itself; the contract is
    |error| <= KAPPA Z E (+ the usual relative tolerance), which here still means better than 1e-4 of D."""
    from oracle import nfs_oracle as o

    W = H = 64
    A, B = 20000.0, 6000.0
    k0x, k0y, w, N = 5, 3, 0.0005, 1200
    x = np.arange(W)[None, :]
    y = np.arange(H)[:, None]
    st = np.stack([np.round(A + B * np.cos(2 * np.pi * (k0x * x / W + k0y * y / H) - w * t)) for t in range(N)]).astype(np.uint16)
    lags = list(range(1, 27)) + [40, 80]
    D, I_q, cnt, D2d, I2d = run(binding, st, lags, 16)
    ref = o.structure_function(st, lags, 16, want_2d=True)
    f = st.astype(np.float64)
    F = np.fft.fft2(f / f.mean(axis=(1, 2), keepdims=True), norm="ortho")[:, k0y, k0x]
    Z, E = np.abs(F - F[0]).max(), np.abs(F[1:] - F[:-1]).max()
    r = ref.D2d[:, k0y, k0x]
    assert Z / E > 1000 and r[0] < 1e-6 * Z * Z                       # the regime the contract is about
    err = np.abs(D2d[:, k0y, k0x] - r)
    assert np.all(err <= KAPPA * Z * E + 1e-5 * r), (err / (Z * E)).max()
    assert (err / r).max() < 1e-4
    # and over the whole half plane the usual rule: relative where D2d is above the threshold, the floor below
    R = ref.D2d[:, :, :W // 2 + 1]
    m = R > 1e-6 * R.max()
    assert (np.abs(D2d - R)[m] / R[m]).max() < TOL_PIXEL
    assert np.abs(D2d - R)[~m].max() <= recurrence_floor(R, lags)
    # NFS_FLAG_DIRECT: the error no longer knows about the excursion Z: a few fp32 roundings of D itself
    _, _, _, D2d_direct, _ = run(binding, st, lags, 16, direct=True)
    err_d = np.abs(D2d_direct[:, k0y, k0x] - r)
    assert (err_d / r).max() < 5e-6, (err_d / r).max()
    assert (np.abs(D2d_direct - R)[m] / R[m]).max() < TOL_PIXEL


def test_travelling_fringe_closed_form(binding):
    """P4/P9: I_t = A + B cos(2 pi k0.x - w t): D2d(k0,tau) = (B/2A)^2 WH (2 - 2 cos w tau), all in one |q| bin."""
    W = H = 64
    A, B = 20000.0, 6000.0
    k0x, k0y, w = 5, 3, 0.37
    x = np.arange(W)[None, :]
    y = np.arange(H)[:, None]
    N = 40
    st = np.stack([np.round(A + B * np.cos(2 * np.pi * (k0x * x / W + k0y * y / H) - w * t)) for t in range(N)])
    lags = [1, 2, 3, 5, 8, 13]
    n_b = 32
    D, I_q, cnt, D2d, I2d = run(binding, st.astype(np.uint16), lags, n_b)
    b0 = int(np.floor(n_b * 2 * np.sqrt((k0x / W) ** 2 + (k0y / H) ** 2)))
    for l, tau in enumerate(lags):
        expect = (B / (2 * A)) ** 2 * W * H * (2 - 2 * np.cos(w * tau))
        assert D2d[l, k0y, k0x] == pytest.approx(expect, rel=2e-3)       # uint16 rounding of the fringe
        # the conjugate mode (-k0) is the other half of the full plane: bin mean = 2 * expect / c_b
        assert D[l, b0] == pytest.approx(2 * expect / cnt[b0], rel=5e-3)
        others = np.delete(D[l], b0)
        assert others.max() < 1e-4 * D[l, b0]


def test_ramp(binding):
    """P6: I_t = I_0 + t G with sum(G) = 0 (constant mean): D2d(k,tau) = tau^2 |F_G(k)|^2 for k != 0."""
    rng = np.random.default_rng(11)
    W = H = 64
    I0 = rng.integers(20000, 30000, size=(H, W))
    G = rng.integers(-20, 21, size=(H, W))
    G.flat[0] -= G.sum()
    st = np.stack([I0 + t * G for t in range(16)]).astype(np.uint16)
    lags = [1, 2, 3, 6]
    D, I_q, cnt, D2d, I2d = run(binding, st, lags, 16)
    FG = np.abs(np.fft.rfft2(G / I0.mean(), norm="ortho")) ** 2
    m = FG > 1e-6 * FG.max()
    m[0, 0] = False
    for l, tau in enumerate(lags):
        assert (np.abs(D2d[l] - tau * tau * FG)[m] / (tau * tau * FG[m])).max() < 1e-4


def test_parseval_and_dc(binding):
    """P2: sum_k D2d(k,tau) over the full plane = < sum_x (i_t - i_{t+tau})^2 >_t ; D2d(DC) = 0 (P3)."""
    cfg = synth.config(0)
    st = synth.make_stack(cfg, "cpu").numpy()
    lags = [1, 4, 8]
    D, I_q, cnt, D2d, I2d = run(binding, st, lags, cfg.n_qbins)
    i = st.astype(np.float64)
    i /= i.mean(axis=(1, 2), keepdims=True)
    n = cfg.W // 2
    wgt = np.full(n + 1, 2.0)
    wgt[0] = wgt[n] = 1.0
    for l, tau in enumerate(lags):
        real = np.mean(((i[:-tau] - i[tau:]) ** 2).sum(axis=(1, 2)))
        four = (D2d[l] * wgt[None, :]).sum()
        assert four == pytest.approx(real, rel=1e-5)
        assert D2d[l, 0, 0] < 1e-9 * D2d[l].max()


# --------------------------------------------------------------------------------------------------------------
# variance form of the fluctuation spectrum: nfs_get_variance / nfs_get_V2d
# --------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("idx,W,N,batch,split", [(0, 64, 32, 0, 0), (1, 128, 300, 0, 0), (1, 256, 700, 128, 100),
                                                 (2, 512, 120, 0, 0), (3, 1024, 40, 16, 0)])
def test_variance_spectrum_against_oracle(binding, oracle, idx, W, N, batch, split):
    n_b = max(8, W // 4)
    lags = [1, 2, 3, 5, 8, 13, 21]
    cfg = synth.config(idx, W=W, N=N, lags=lags, n_qbins=n_b)
    st = synth.make_stack(cfg, "cuda")
    ref = oracle.variance_spectrum(st.cpu().numpy(), n_b, want_2d=True)
    nfs = binding.NFS(W, W, lags, n_b, batch_frames=batch)
    if split:
        for i in range(0, N, split):
            nfs.push(st[i:i + split].contiguous())
    else:
        nfs.push(st)
    V = nfs.variance()
    V2d = nfs.V2d()
    D, I_q, cnt = nfs.finalize()
    assert np.array_equal(V, nfs.variance()), "a snapshot: asking twice changes nothing"
    nfs.close()
    nz = ref.counts > 0
    assert np.array_equal(cnt, ref.counts)
    assert np.all(V[~nz] == 0.0)
    eV = float(np.max(np.abs(V[nz] - ref.V_q[nz]) / ref.V_q[nz]))
    assert eV < 1e-4, "binned V rel err %.3e" % eV
    r2 = ref.V2d[:, :W // 2 + 1]
    m = r2 > 1e-6 * r2.max()
    eP = float(np.max(np.abs(V2d[m] - r2[m]) / r2[m]))
    assert eP < 1e-3, "per-pixel V2d rel err %.3e" % eP
    assert V2d[0, 0] < 1e-9 * r2.max()          # every normalised frame has the same DC value
    # for long lags the difference spectrum approaches twice the variance, never far above it
    assert np.all(D[-1][nz] < 4.0 * V[nz] * 1.01 + 1e-30)


def test_variance_of_a_constant_stack_vanishes(binding):
    one = torch.randint(100, 4000, (64, 64), dtype=torch.int32, device="cuda").to(torch.uint16)
    st = one[None].repeat(20, 1, 1).contiguous()
    nfs = binding.NFS(64, 64, [1, 2], 16)
    nfs.push(st)
    # F'_t = FFT(i_t - r) is the same tiny rounding residual for every frame; what is left of its variance is the
    # rounding of the sums (the oracle's two-pass form leaves < 1e-25 as well), against fluctuation spectra of order 1e-4
    assert np.all(nfs.variance() < 1e-18) and np.all(nfs.V2d() < 1e-18)
    nfs.close()


def test_all_lags_identity_ties_D_to_the_variance_on_the_gpu(binding, oracle):
    """The paper's own case (all N - 1 lags, N(N-1)/2 pairs) at reduced size: every lag 1..N-1 in
    one context (16 lag groups), parity with the oracle, and the identity sum_tau (N - tau) D2d(k,tau) = N^2 V2d(k)
    between two outputs that come from different accumulators (pair totals vs. the I sums)."""
    W, N, n_b = 64, 200, 16
    lags = list(range(1, N))
    cfg = synth.config(1, W=W, N=N, lags=lags, n_qbins=n_b)
    st = synth.make_stack(cfg, "cuda")
    nfs = binding.NFS(W, W, lags, n_b)
    nfs.push(st)
    D, I_q, cnt = nfs.finalize()
    V2d = nfs.V2d()
    V = nfs.variance()
    acc = np.zeros_like(V2d)
    for l, tau in enumerate(lags):
        acc += (N - tau) * nfs.D2d(l)
    nfs.close()
    m = V2d > 1e-6 * V2d.max()
    assert np.max(np.abs(acc[m] / N ** 2 - V2d[m]) / V2d[m]) < 2e-5
    ref = oracle.structure_function(st.cpu().numpy(), lags, n_b)
    nz = ref.counts > 0
    assert np.array_equal(cnt, ref.counts)
    assert np.max(np.abs(D[:, nz] - ref.D[:, nz]) / ref.D[:, nz]) < 1e-4
    lhs = sum((N - tau) * D[l] for l, tau in enumerate(lags)) / N ** 2
    assert np.max(np.abs(lhs[nz] - V[nz]) / V[nz]) < 2e-5
