"""Seeded synthetic shadowgraph stacks (input generator only — none of the method's arithmetic).

Stands in for the paper's unpublished camera stacks (beam-dominated static image,
residual fringes, weak diffusing fluctuations, 4 Hz).  Recipe: SURVEY.md §8(d) / DESIGN.md §4,
values fixed by BASELINE.json `configs`:

  frame_t = clip(round(A * E * prod_j[1 + 0.05 cos(2 pi (kjx x/W + kjy y/H) + phi_j)] * (1 + delta_t)
                       -> optional Poisson -> + N(0, 5^2) read noise), 0, 2^bits - 1)  as uint16
  E       = exp(-((x-(W-1)/2)^2 + (y-(H-1)/2)^2) / (2 sigma_b^2))
  delta_t = delta_rms * (WH / sqrt(sum_full S^2)) * irfft2(a_t),   a_t an Ornstein-Uhlenbeck process
            per Fourier mode: a_0 = S xi, a_{t+1} = a_t e^{-Gamma} + S sqrt(1 - e^{-2 Gamma}) xi,
            S(q) = 1/(1 + (q/q0)^4), S(0) = 0, Gamma(q) = gamma0 (q/q0)^2, q in cycles/px.

This module (harness code at the repo root, outside the product package) serves both the CUDA path's
tests/bench and the oracle's tests; it imports neither.
It is harness code: torch (incl. torch.fft) is used so configs 2-4 can be generated on the GPU.
Oracle and library always consume the *same uint16 bytes* within a run.
"""
from dataclasses import dataclass, field, replace
from typing import List, Tuple

import math

import torch


def log_lags(n: int = 40, tmax: int = 500) -> List[int]:
    """tau_i = max(tau_{i-1}+1, round(tmax^(i/(n-1))))  (config 3)"""
    out: List[int] = []
    for i in range(n):
        v = int(round(tmax ** (i / (n - 1))))
        out.append(max(v, out[-1] + 1) if out else max(v, 1))
    return out


@dataclass
class StackConfig:
    name: str
    W: int
    H: int
    N: int
    lags: List[int]
    n_qbins: int
    sigma_b: float
    q0: float
    gamma0: float
    A: float
    bits: int
    poisson: bool
    n_random_fringes: int
    seed: int
    delta_rms: float = 0.02
    read_noise: float = 5.0
    chunk: int = 0  # config 4: frames per streamed chunk (0 = caller's choice)
    fringes: List[Tuple[float, float, float]] = field(default_factory=list)  # filled by SynthStack


def config(idx: int, W: int = 0, N: int = 0, lags=None, n_qbins: int = 0) -> StackConfig:
    """BASELINE.json configs[idx]; W/N/lags/n_qbins override for scaled-down parity cases
    (sigma_b and q0 keep their ratio to the frame size)."""
    base = {
        0: dict(W=64, N=32, lags=list(range(1, 9)), n_qbins=32, q0W=6.4, gamma0=0.05, A=2000.0, bits=16,
                poisson=False, nrf=0, chunk=0),
        1: dict(W=512, N=1000, lags=list(range(1, 101)), n_qbins=128, q0W=10.24, gamma0=0.05, A=2000.0, bits=12,
                poisson=False, nrf=0, chunk=0),
        2: dict(W=1024, N=2000, lags=list(range(1, 101)), n_qbins=256, q0W=10.24, gamma0=0.01, A=8000.0, bits=14,
                poisson=True, nrf=0, chunk=0),
        3: dict(W=2048, N=1000, lags=log_lags(40, 500), n_qbins=512, q0W=10.24, gamma0=0.05, A=8000.0, bits=14,
                poisson=True, nrf=3, chunk=0),
        4: dict(W=1024, N=10000, lags=list(range(1, 1001)), n_qbins=256, q0W=10.24, gamma0=0.01, A=8000.0, bits=14,
                poisson=True, nrf=0, chunk=256),
        # not a BASELINE.json config: the workload of the paper's only timing (Fig. 3: 512 x 512 px,
        # N = 2048 images, all N - 1 = 2047 lags, full 2-D spectra kept), generator of config 1
        5: dict(W=512, N=2048, lags=list(range(1, 2048)), n_qbins=128, q0W=10.24, gamma0=0.05, A=2000.0, bits=12,
                poisson=False, nrf=0, chunk=0),
    }[idx]
    w = W or base["W"]
    return StackConfig(
        name=("config%d" % idx if idx < 5 else "paper-fig3") if not (W or N or lags or n_qbins) else "config%d-scaled" % idx,
        W=w, H=w, N=N or base["N"], lags=list(lags) if lags is not None else base["lags"],
        n_qbins=n_qbins or base["n_qbins"], sigma_b=0.3125 * w, q0=base["q0W"] / w, gamma0=base["gamma0"],
        A=base["A"], bits=base["bits"], poisson=base["poisson"], n_random_fringes=base["nrf"], seed=idx,
        chunk=base["chunk"])


class SynthStack:
    """Sequential generator: `next_frames(n)` returns the next n frames, uint16 [n][H][W] on `device`."""

    def __init__(self, cfg: StackConfig, device="cpu"):
        self.cfg = cfg
        self.device = torch.device(device)
        self.gen = torch.Generator(device=self.device)
        self.gen.manual_seed(1000003 * cfg.seed + 12345)
        W, H = cfg.W, cfg.H
        dev, f32 = self.device, torch.float32
        x = torch.arange(W, device=dev, dtype=f32)
        y = torch.arange(H, device=dev, dtype=f32)
        E = torch.exp(-(((x - (W - 1) / 2) ** 2)[None, :] + ((y - (H - 1) / 2) ** 2)[:, None]) / (2 * cfg.sigma_b ** 2))
        fr = [(W / 8.0, H / 16.0, 0.0)]
        if cfg.n_random_fringes:
            u = torch.rand(cfg.n_random_fringes, 3, generator=self.gen, device=dev).cpu().tolist()
            for a, b, c in u:
                fr.append((float(round(W / 16 + a * (W / 4 - W / 16))), float(round(-H / 4 + b * H / 2)), 2 * math.pi * c))
        cfg = replace(cfg, fringes=fr)
        self.cfg = cfg
        static = cfg.A * E
        for kx, ky, ph in fr:
            static = static * (1 + 0.05 * torch.cos(2 * math.pi * (kx * x[None, :] / W + ky * y[:, None] / H) + ph))
        self.static = static
        kxh = torch.arange(W // 2 + 1, device=dev, dtype=f32) / W
        kyf = torch.arange(H, device=dev, dtype=f32)
        kyf = torch.where(kyf < H // 2, kyf, kyf - H) / H
        q = torch.sqrt(kxh[None, :] ** 2 + kyf[:, None] ** 2)
        S = 1.0 / (1.0 + (q / cfg.q0) ** 4)
        S[0, 0] = 0.0
        wgt = torch.full_like(S, 2.0)
        wgt[:, 0] = 1.0
        wgt[:, -1] = 1.0
        self.S = S
        self.amp = cfg.delta_rms * (W * H) / math.sqrt(float((wgt * S * S).sum()))
        G = cfg.gamma0 * (q / cfg.q0) ** 2
        self.decay = torch.exp(-G)
        self.kick = S * torch.sqrt(1 - torch.exp(-2 * G))
        self.a = None
        self.t = 0

    def _xi(self):
        W, H = self.cfg.W, self.cfg.H
        r = torch.randn(2, H, W // 2 + 1, generator=self.gen, device=self.device)
        return torch.complex(r[0], r[1]) * (1 / math.sqrt(2.0))

    def next_frames(self, n: int) -> torch.Tensor:
        cfg = self.cfg
        modes = []
        for _ in range(n):
            if self.a is None:
                self.a = self.S * self._xi()
            else:
                self.a = self.a * self.decay + self.kick * self._xi()
            modes.append(self.a)
            self.t += 1
        delta = self.amp * torch.fft.irfft2(torch.stack(modes), s=(cfg.H, cfg.W))
        img = self.static[None] * (1 + delta)
        if cfg.poisson:
            img = torch.poisson(img.clamp_min(0), generator=self.gen)
        img = img + cfg.read_noise * torch.randn(img.shape, generator=self.gen, device=self.device)
        return torch.round(img).clamp_(0, 2 ** cfg.bits - 1).to(torch.uint16)


def make_stack(cfg: StackConfig, device="cpu", n: int = 0, chunk: int = 64) -> torch.Tensor:
    """Whole stack [N][H][W] uint16 on `device` (generated in chunks to bound temporaries)."""
    s = SynthStack(cfg, device)
    n = n or cfg.N
    out = torch.empty((n, cfg.H, cfg.W), dtype=torch.uint16, device=s.device)
    for i in range(0, n, chunk):
        m = min(chunk, n - i)
        out[i:i + m] = s.next_frames(m)
    return out
