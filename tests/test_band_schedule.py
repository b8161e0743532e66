"""The out-of-core band schedule ("N - 1 = alpha N* + beta ... first triangle ... alpha diagonals ...
upper-right triangle", Fig. 2(b) L37): host logic without a GPU (transfer counts against the
paper's closed form N_FFT = N (2 alpha - 3 + 2 / alpha)), and on the GPU the result of a small stack forced to three
bands against the CPU oracle and against the in-memory schedule."""
import numpy as np
import pytest

import synth
from paper_1209_3362_b200 import binding


def n_fft_paper(N, alpha):
    """image transfers to the G-RAM for beta = 0."""
    return N * (2 * alpha - 3 + 2.0 / alpha)


def paper_schedule_uploads(N, n_star, alpha):
    """The schedule as PAPER.md:L33 words it, counted literally: every image enters the G-RAM once while the first
    triangle (lags <= N*) is processed; every further diagonal band is a sweep of N - N* steps, each of which replaces
    one FIFO image and uploads one 'current image'."""
    uploads = N
    for _ in range(2, alpha + 1):
        uploads += 2 * (N - n_star)
    return uploads


@pytest.mark.parametrize("alpha,n_star", [(2, 50), (3, 50), (4, 32), (8, 16)])
def test_transfer_count_against_paper_formula(alpha, n_star):
    N = alpha * n_star          # the paper's simplification: beta = 0 and N - 1 ~ N
    # R17: the literal count of the paper's schedule is its closed form
    assert paper_schedule_uploads(N, n_star, alpha) == pytest.approx(n_fft_paper(N, alpha), abs=1e-9)
    lags = list(range(1, N))    # all N - 1 lags
    b = 8
    plan = binding.nfs_band_plan(N, lags, n_star + 2 * b, b)
    assert plan["band_width"] == n_star and plan["batch"] == b
    assert plan["bands"] == -(-(N - 1) // n_star) == alpha
    # this schedule: band k (lags (k N*, (k+1) N*]) uploads every OLD frame 0 .. N-1-tmin and every NEW frame tmin .. N-1 once
    expect = sum(N - (k * n_star + 1) for k in range(1, alpha))
    assert plan["old_uploads"] == expect and plan["new_uploads"] == expect
    ours = N + plan["old_uploads"] + plan["new_uploads"]   # + the N frames of the streaming pass
    assert ours <= n_fft_paper(N, alpha)                   # a band stops where its pairs end; the paper sweeps N - N* steps
    if alpha == 2:
        assert abs(ours - n_fft_paper(N, alpha)) <= 2
    # far fewer transfers than frame pairs (the paper's point: 2 alpha N << N^2 / 2)
    assert ours < 2 * alpha * N and (alpha <= 4 or ours < N * (N - 1) // 2)


def test_band_plan_edges():
    # everything fits: one band, nothing is uploaded again
    p = binding.nfs_band_plan(100, list(range(1, 41)), 40 + 2 * 16, 16)
    assert p["bands"] == 1 and p["old_uploads"] == p["new_uploads"] == p["launches"] == 0
    # sparse lags: a band without requested lags costs nothing; a band beyond the stack costs nothing
    p = binding.nfs_band_plan(60, [1, 2, 3, 120, 121], 20 + 2 * 4, 4)
    assert p["bands"] == 7 and p["old_uploads"] == 0 and p["launches"] == 0
    p = binding.nfs_band_plan(200, [1, 2, 3, 120, 121], 20 + 2 * 4, 4)
    assert p["old_uploads"] == p["new_uploads"] == (200 - 120) + (200 - 121)   # lag 120 closes band 5, lag 121 opens band 6
    with pytest.raises(binding.NFSError):
        binding.nfs_band_plan(100, [30, 31], 20 + 8, 4)      # the smallest lag must lie in band 0
    with pytest.raises(binding.NFSError):
        binding.nfs_band_plan(100, [1, 2], 8, 4)             # no room for a band


def test_plan_groups_never_straddle_bands():
    """Through nfs_plan_lags nothing changes (no band width): the banded plan is exercised on the GPU below; here the
    band arithmetic of nfs_band_plan for lags that are not multiples of the band width."""
    p = binding.nfs_band_plan(151, list(range(1, 151)), 50 + 2 * 26, 26)
    assert (p["bands"], p["band_width"], p["batch"]) == (3, 50, 26)
    assert p["old_uploads"] == (151 - 51) + (151 - 101) and p["launches"] == 4 + 2


@pytest.mark.gpu
@pytest.mark.parametrize("lags,cap,batch", [(list(range(1, 151)), 50 + 2 * 26, 26),
                                            ([1, 2, 3, 4, 5, 9, 17, 30, 31, 32, 33, 60, 61, 90, 120, 149], 40 + 2 * 13, 13)])
def test_banded_equals_oracle_and_in_memory(oracle, lags, cap, batch):
    import torch

    assert torch.cuda.is_available()
    cfg = synth.config(0, N=200, lags=lags, n_qbins=24)
    st = synth.make_stack(cfg, "cuda")
    ref = oracle.structure_function(st.cpu().numpy(), lags, cfg.n_qbins)
    plain = binding.NFS(cfg.W, cfg.H, lags, cfg.n_qbins)
    plain.push(st)
    D0, I0, c0 = plain.finalize()
    D2d0 = plain.D2d(len(lags) - 1)
    plain.close()

    nfs = binding.NFS(cfg.W, cfg.H, lags, cfg.n_qbins, batch_frames=batch, ring_frames_cap=cap, max_frames=cfg.N)
    assert nfs.ring_capacity == cap - batch            # the FIFO: a band's window plus a batch
    tc = nfs.transfer_counts()
    assert tc["bands"] >= 3 and tc["band_width"] == cap - 2 * batch
    for i in range(0, 120, 40):
        nfs.push(st[i:i + 40])
    D_a, _, _ = nfs.finalize()                          # snapshot after 120 frames: the sweeps run, the ring is overwritten
    ref_a = oracle.structure_function(st[:120].cpu().numpy(), lags, cfg.n_qbins)
    nfs.push(st[120:])                                  # ... and restored from the host store
    D, I_q, cnt = nfs.finalize()
    D2d = nfs.D2d(len(lags) - 1)
    tc = nfs.transfer_counts()
    pl_a = binding.nfs_band_plan(120, lags, cap, batch)
    pl = binding.nfs_band_plan(cfg.N, lags, cap, batch)
    nfs.close()

    nz = ref.counts > 0
    rows_a = ref_a.n_pairs > 0
    assert np.array_equal(cnt, ref.counts)
    assert np.max(np.abs(D_a[rows_a][:, nz] - ref_a.D[rows_a][:, nz]) / ref_a.D[rows_a][:, nz]) < 1e-4
    assert np.all(D_a[~rows_a] == 0.0)
    assert np.max(np.abs(D[:, nz] - ref.D[:, nz]) / ref.D[:, nz]) < 1e-4
    assert np.max(np.abs(I_q[nz] - ref.I_q[nz]) / ref.I_q[nz]) < 1e-4
    assert np.max(np.abs(D[:, nz] - D0[:, nz]) / D0[:, nz]) < 1e-5   # same result as the in-memory schedule
    assert np.max(np.abs(I_q[nz] - I0[nz]) / I0[nz]) < 1e-6 and np.array_equal(cnt, c0)   # other batch boundaries: fp32 rounding only
    m = D2d0 > 1e-6 * D2d0.max()
    assert np.max(np.abs(D2d[m] - D2d0[m]) / D2d0[m]) < 1e-5
    # transfers: every frame downloaded once; uploads = the two walks + the ring restored before the second push
    assert tc["d2h_frames"] == cfg.N
    restored = min(120, cap - batch)
    assert tc["h2d_frames"] == pl_a["old_uploads"] + pl_a["new_uploads"] + restored + pl["old_uploads"] + pl["new_uploads"]
