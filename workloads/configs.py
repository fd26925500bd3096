"""Seeded synthetic PWA workloads shaped like BASELINE.json's `configs`.

The paper fits its own generated psi(3686) -> phi K+ K- sample (§3), which is not
available; these workloads stand in for it: a handful to a hundred resonances with floating mass
and width in the range of Table 1, N_MC >> N_Data, two or
more incoherent components (the sum over mu in Eq. 1).

What is generated (layouts are the ones `include/pwa.h` takes):
  theta_true[4R]   (a, phi, M, Gamma) per resonance: a~U[0.5,1.5], phi~U[-pi,pi], M~U[0.5,2.8], Gamma~U[0.02,0.4]
  res_chan[R]      r mod C
  mass[C][N]       config 1: m~U[0.3,3.0]; others: (s12,s13) uniform in a Dalitz-like triangle, m=sqrt(s)
  amp[R][H][N][2]  Re,Im ~ N(0,1) iid
  weight[N_data]   config 3 only, U[0.5,1.5]
  data events      accept-reject on candidates drawn like MC events, kept in candidate order

The accept-reject step has to look at an intensity to decide which candidates to keep.  That
decision is workload shaping, not part of the likelihood evaluation under test: `_shaping_intensity`
below is used for nothing else, neither the oracle nor the CUDA path imports it, and both always
consume the finished arrays, so a mistake here would change the input distribution and never the
parity between the two.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace
from typing import Optional

import torch

from . import rng

# stream ids
S_THETA, S_MC_MASS, S_MC_F, S_CAND_MASS, S_CAND_F, S_ACCEPT, S_WEIGHT, S_V, S_START = range(9)

S_MIN = 0.09          # GeV^2, lower edge of every Dalitz variable (m >= 0.3 GeV)
S_TOT = 9.18          # GeV^2, s12 + s13 + s23
M_LO, M_HI = 0.3, 3.0  # GeV, config 1 mass window


@dataclass(frozen=True)
class Config:
    name: str
    index: int
    n_res: int
    n_hel: int
    n_chan: int
    n_mc: int
    n_data: int
    weighted: bool = False
    dalitz: bool = True
    table1: bool = False       # take (M, Gamma) from the paper's Table 1 instead of the uniform draw

    @property
    def seed(self) -> int:
        return 20240315 + self.index

    @property
    def n_par(self) -> int:
        return 4 * self.n_res

    def bytes_per_event(self, data: bool) -> int:
        """Algorithmic HBM bytes one evaluation must read per event."""
        return 16 * self.n_res * self.n_hel + 8 * self.n_chan + (8 if (data and self.weighted) else 0)

    def bytes_per_eval(self) -> int:
        return self.n_mc * self.bytes_per_event(False) + self.n_data * self.bytes_per_event(True)

    def scaled(self, n_mc: int, n_data: int) -> "Config":
        """Same model, fewer events (parity-test sizes)."""
        return replace(self, n_mc=n_mc, n_data=n_data)


# BASELINE.json `configs` 1-4 (config 5 = a fit on config 2's arrays) and a paper-shaped extra.
CONFIGS = {
    1: Config("tiny", 1, n_res=2, n_hel=2, n_chan=1, n_mc=50_000, n_data=10_000, dalitz=False),
    2: Config("medium", 2, n_res=10, n_hel=3, n_chan=2, n_mc=1_000_000, n_data=100_000),
    3: Config("large", 3, n_res=30, n_hel=2, n_chan=3, n_mc=5_000_000, n_data=500_000, weighted=True),
    4: Config("big", 4, n_res=100, n_hel=4, n_chan=3, n_mc=10_000_000, n_data=1_000_000),
    # PAPER.md:102-113 (Table 1), :141: six resonances, two incoherent components, 10 000 data events,
    # 1 M integration events; one K+K- mass channel.
    6: Config("paper_shape", 6, n_res=6, n_hel=2, n_chan=1, n_mc=1_000_000, n_data=10_000,
              dalitz=False, table1=True),
}

# PAPER.md:106-113 (Table 1): mass and width in GeV, in the table's row order.
TABLE1_M_GAMMA = [(1.022, 0.209), (2.545, 0.303), (1.522, 0.091), (1.672, 0.169), (1.302, 0.189), (2.150, 0.143)]


@dataclass
class Workload:
    cfg: Config
    theta_true: torch.Tensor             # [4R] fp64, CPU
    res_chan: torch.Tensor               # [R] int32, CPU
    mc_mass: torch.Tensor                # [C][N_mc]
    mc_amp: torch.Tensor                 # [R][H][N_mc][2]
    data_mass: torch.Tensor              # [C][N_data]
    data_amp: torch.Tensor               # [R][H][N_data][2]
    data_weight: Optional[torch.Tensor]  # [N_data] or None
    info: dict = field(default_factory=dict)


def theta_true(cfg: Config) -> torch.Tensor:
    R = cfg.n_res
    key = lambda k: rng.stream_key(cfg.seed, S_THETA, k)
    th = torch.empty(R, 4, dtype=torch.float64)
    th[:, 0] = rng.uniform(key(0), 0, R, 0.5, 1.5)
    th[:, 1] = rng.uniform(key(1), 0, R, -math.pi, math.pi)
    th[:, 2] = rng.uniform(key(2), 0, R, 0.5, 2.8)
    th[:, 3] = rng.uniform(key(3), 0, R, 0.02, 0.4)
    if cfg.table1:
        th[:, 2:4] = torch.tensor(TABLE1_M_GAMMA[:R], dtype=torch.float64)
    return th.reshape(-1)


def random_start(cfg: Config, k: int) -> torch.Tensor:
    """k-th seeded fit starting point: a~U[0.1,2], phi~U[-pi,pi], M~U[0.5,2.8], Gamma~U[0.02,0.4]."""
    R = cfg.n_res
    key = lambda j: rng.stream_key(cfg.seed, S_START, 4 * k + j)
    th = torch.empty(R, 4, dtype=torch.float64)
    th[:, 0] = rng.uniform(key(0), 0, R, 0.1, 2.0)
    th[:, 1] = rng.uniform(key(1), 0, R, -math.pi, math.pi)
    th[:, 2] = rng.uniform(key(2), 0, R, 0.5, 2.8)
    th[:, 3] = rng.uniform(key(3), 0, R, 0.02, 0.4)
    return th.reshape(-1)


def direction(cfg: Config, k: int = 0) -> torch.Tensor:
    """k-th seeded HVP direction v ~ N(0,1)^P."""
    a, _ = rng.normal_pair(cfg.seed, S_V, k, 0, cfg.n_par)
    return a


def res_chan(cfg: Config) -> torch.Tensor:
    return (torch.arange(cfg.n_res, dtype=torch.int64) % cfg.n_chan).to(torch.int32)


def masses(cfg: Config, stream: int, start: int, count: int, device="cpu") -> torch.Tensor:
    """mass[C][count] for events start..start+count-1 of the given stream."""
    seed = cfg.seed
    if not cfg.dalitz:
        assert cfg.n_chan == 1
        return rng.uniform(rng.stream_key(seed, stream, 0), start, count, M_LO, M_HI, device).reshape(1, count)
    u1 = rng.uniform01(rng.stream_key(seed, stream, 0), start, count, device)
    u2 = rng.uniform01(rng.stream_key(seed, stream, 1), start, count, device)
    flip = (u1 + u2) > 1.0
    u1 = torch.where(flip, 1.0 - u1, u1)
    u2 = torch.where(flip, 1.0 - u2, u2)
    side = S_TOT - 3.0 * S_MIN
    s12 = S_MIN + side * u1
    s13 = S_MIN + side * u2
    s23 = S_TOT - s12 - s13
    return torch.sqrt(torch.stack([s12, s13, s23][: cfg.n_chan], dim=0))


def fill_amp(cfg: Config, stream: int, start: int, count: int, out: torch.Tensor, out_start: int = 0) -> None:
    """Write amp[r][h][out_start:out_start+count][:] for events start..start+count-1 of `stream`."""
    dev = out.device
    for r in range(cfg.n_res):
        for h in range(cfg.n_hel):
            re, im = rng.normal_pair(cfg.seed, stream, r * cfg.n_hel + h, start, count, dev)
            out[r, h, out_start:out_start + count, 0] = re
            out[r, h, out_start:out_start + count, 1] = im


def _shaping_intensity(theta, rchan, mass, amp):
    """Intensity used ONLY to accept or reject data candidates (see the module docstring)."""
    th = theta.to(mass.device).reshape(-1, 4)
    a, phi, M, G = th[:, 0], th[:, 1], th[:, 2], th[:, 3]
    m = mass[rchan.to(mass.device).long()]                                   # [R][n]
    z = torch.polar(a, phi)[:, None] / torch.complex((M * M)[:, None] - m * m, (-M * G)[:, None].expand_as(m))
    A = (z[:, None, :] * torch.view_as_complex(amp)).sum(dim=0)              # [H][n]
    return (A.real ** 2 + A.imag ** 2).sum(dim=0)


def make_workload(cfg: Config, device="cpu", chunk: int = 1 << 18, imax_events: int = 1_000_000,
                  max_candidates: int = 2_000_000_000) -> Workload:
    """Generate the full workload of `cfg` on `device` (CPU for test sizes, the GPU for full sizes)."""
    dev = torch.device(device)
    R, H, C = cfg.n_res, cfg.n_hel, cfg.n_chan
    th = theta_true(cfg)
    rc = res_chan(cfg)

    mc_mass = torch.empty(C, cfg.n_mc, dtype=torch.float64, device=dev)
    mc_amp = torch.empty(R, H, cfg.n_mc, 2, dtype=torch.float64, device=dev)
    imax = 0.0
    for s in range(0, cfg.n_mc, chunk):
        n = min(chunk, cfg.n_mc - s)
        mc_mass[:, s:s + n] = masses(cfg, S_MC_MASS, s, n, dev)
        fill_amp(cfg, S_MC_F, s, n, mc_amp, s)
        if s < imax_events:
            k = min(n, imax_events - s)
            imax = max(imax, float(_shaping_intensity(th, rc, mc_mass[:, s:s + k], mc_amp[:, :, s:s + k]).max()))
    imax *= 1.5

    data_mass = torch.empty(C, cfg.n_data, dtype=torch.float64, device=dev)
    data_amp = torch.empty(R, H, cfg.n_data, 2, dtype=torch.float64, device=dev)
    cand_amp = torch.empty(R, H, chunk, 2, dtype=torch.float64, device=dev)
    kept, tried = 0, 0
    k_acc = rng.stream_key(cfg.seed, S_ACCEPT, 0)
    while kept < cfg.n_data:
        if tried >= max_candidates:
            raise RuntimeError("accept-reject did not fill the data sample")
        cm = masses(cfg, S_CAND_MASS, tried, chunk, dev)
        fill_amp(cfg, S_CAND_F, tried, chunk, cand_amp, 0)
        inten = _shaping_intensity(th, rc, cm, cand_amp)
        u = rng.uniform01(k_acc, tried, chunk, dev)
        idx = torch.nonzero(u * imax < inten).reshape(-1)[: cfg.n_data - kept]
        n = int(idx.numel())
        data_mass[:, kept:kept + n] = cm[:, idx]
        data_amp[:, :, kept:kept + n] = cand_amp[:, :, idx]
        kept += n
        # candidates are consumed whole chunks at a time; the sample is the first n_data accepted
        # candidates in candidate order, whatever the chunk size
        tried += chunk
    del cand_amp

    w = None
    if cfg.weighted:
        w = rng.uniform(rng.stream_key(cfg.seed, S_WEIGHT, 0), 0, cfg.n_data, 0.5, 1.5, dev)
    return Workload(cfg, th, rc, mc_mass, mc_amp, data_mass, data_amp, w,
                    info={"imax": imax, "candidates_tried": tried})
