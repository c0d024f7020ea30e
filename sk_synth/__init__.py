"""Seeded synthetic CHIME-shaped inputs for the SK hot path.

This module is shared by the tests, bench.py and smoke(): it produces the byte buffers that BOTH
the CUDA path and the CPU oracle consume.  It holds none of the SK arithmetic (no decode, no power,
no S1/S2, no SK): it only draws Gaussian noise, adds the interference signals of BASELINE.json's
five configs, and quantises to the 4+4-bit offset encoding of PAPER.md:278 ("4+4-bit complex
Gaussian data (bounded between -7 and 7)"; bit layout from BASELINE.json: high nibble = re + 8,
low nibble = im + 8).

One function here IS part of a method the paper describes: `digitiser_thresholds` turns a
per-receiver sigma into the 14 cumulative thresholds of App. B's round-and-clip digitiser
(PAPER.md:278).  Both simulators (the oracle's and the device's) take that table as an INPUT, the
way they take a seed; neither computes it.  It is pinned on its own, against an erf model written
out in the test (tests/test_oracle_pins.py::test_sim_digitised_layout_and_pmf), so a mistake in it
cannot hide behind the two sides agreeing with each other.

The paper measured on CHIME / Pathfinder sky data, which is not available here;
these buffers take its shapes (2048 / 256 inputs, M = 256, 4+4-bit) and stand in for it.
The recipe is written out in DESIGN.md ("Input recipe").

Noise comes from torch's generator of the chosen device, seeded per chunk of time rows, so a
buffer is reproducible per device type; per-input parameters (sigma_e, phases) always come from a
CPU generator and are identical on every device.  Parity never depends on cross-device equality:
the same bytes are always handed to both sides.
"""
from dataclasses import dataclass, field, replace
from typing import Optional, Tuple

import math

import torch

BASE_SEED = 181810365  # + config index


@dataclass(frozen=True)
class SKConfig:
    name: str
    index: int
    E: int
    F: int
    T: int
    M: int
    n_sigma: float = 3.0
    sigma: Tuple[float, float] = (2.5, 2.5)      # per-input sigma ~ U[lo, hi] per component
    # interference (all optional)
    cw_block_inputs: Optional[Tuple[int, int, int]] = None   # (block, first input, n inputs), f = 0
    cw_freqs: Tuple[int, ...] = ()                # CW on all inputs, all time, f % cw_period in set
    cw_period: int = 0
    cw_amp: float = 4.0
    cw_cycles_per_sample: float = 0.0371
    burst_fraction: float = 0.0                   # fraction of blocks holding one 8-sample pulse
    burst_len: int = 8
    burst_amp: float = 6.0
    sine_freqs: Tuple[int, ...] = ()              # strong sinusoid on the first sine_inputs inputs
    sine_inputs: int = 0
    sine_amp: float = 6.0
    sine_cycles_per_sample: float = 0.0913
    note: str = ""

    @property
    def seed(self) -> int:
        return BASE_SEED + self.index

    @property
    def B(self) -> int:
        return self.T // self.M

    @property
    def nbytes(self) -> int:
        return self.T * self.F * self.E

    def with_(self, **kw) -> "SKConfig":
        return replace(self, **kw)


CONFIGS = (
    SKConfig("cfg0_pathfinder_toy", 0, E=256, F=1, T=4096, M=256, sigma=(2.5, 2.5),
             cw_block_inputs=(7, 0, 32),
             note="E=256 toy, CW amp 4 on inputs 0-31 during block 7, N=256, 3 sigma"),
    SKConfig("cfg1_chime_frame", 1, E=2048, F=1, T=49152, M=256, sigma=(1.5, 3.5),
             note="one CHIME frequency frame, pure noise, per-input sigma ~ U[1.5,3.5]"),
    SKConfig("cfg2_rfi_mix", 2, E=2048, F=16, T=32768, M=256, sigma=(1.5, 3.5),
             cw_freqs=(2, 7, 11), cw_period=16, burst_fraction=0.05,
             sine_freqs=(13,), sine_inputs=64,
             note="CW in f=2,7,11; 8-sample amp-6 bursts in 5% of blocks; sinusoid on 64 inputs of f=13"),
    SKConfig("cfg3_sweep", 3, E=2048, F=4, T=65536, M=256, sigma=(2.5, 2.5),
             note="sigma=2.5 noise; swept over M and N by the caller"),
    SKConfig("cfg4_streaming", 4, E=2048, F=64, T=65536, M=256, sigma=(1.5, 3.5),
             cw_freqs=(2, 7, 11), cw_period=16, burst_fraction=0.05,
             sine_freqs=(13, 29, 45, 61), sine_inputs=64,
             note="config 2's mix scaled to 64 frequencies (~20% of cells carry RFI), 8 GiB"),
)


def config(i: int) -> SKConfig:
    return CONFIGS[i]


def _cpu_gen(seed: int) -> torch.Generator:
    g = torch.Generator(device="cpu")
    g.manual_seed(seed)
    return g


def sigma_per_input(cfg: SKConfig, seed_offset: int = 0) -> torch.Tensor:
    """float64 [E], per-component noise sigma of each input (CPU generator: device independent)."""
    lo, hi = cfg.sigma
    if lo == hi:
        return torch.full((cfg.E,), float(lo), dtype=torch.float64)
    u = torch.rand(cfg.E, generator=_cpu_gen(cfg.seed * 7919 + 1 + seed_offset), dtype=torch.float64)
    return lo + (hi - lo) * u


def _phases(cfg: SKConfig, tag: int, shape) -> torch.Tensor:
    u = torch.rand(shape, generator=_cpu_gen(cfg.seed * 7919 + 100 + tag), dtype=torch.float64)
    return 2.0 * math.pi * u


def burst_starts(cfg: SKConfig) -> torch.Tensor:
    """int64 [n]: absolute start sample of each 8-sample pulse (one per chosen block)."""
    if cfg.burst_fraction <= 0:
        return torch.zeros(0, dtype=torch.int64)
    g = _cpu_gen(cfg.seed * 7919 + 200)
    n = max(1, int(round(cfg.burst_fraction * cfg.B)))
    blocks = torch.randperm(cfg.B, generator=g)[:n].sort().values
    off = torch.randint(0, cfg.M - cfg.burst_len + 1, (n,), generator=g)
    return blocks * cfg.M + off


def rfi_cells(cfg: SKConfig, include_sine: bool = True) -> torch.Tensor:
    """bool [B][F]: cells into which the recipe injects interference (for reporting only).
    include_sine=False leaves out cells whose only interference is the sinusoid confined to a few
    inputs (it moves the full-array SK by only a few sigma)."""
    m = torch.zeros(cfg.B, cfg.F, dtype=torch.bool)
    if cfg.cw_block_inputs is not None:
        m[cfg.cw_block_inputs[0], 0] = True
    for f in range(cfg.F):
        if cfg.cw_period and (f % cfg.cw_period) in cfg.cw_freqs:
            m[:, f] = True
        if include_sine and f in cfg.sine_freqs and cfg.sine_inputs:
            m[:, f] = True
    st = burst_starts(cfg)
    if st.numel():
        m[st // cfg.M, :] = True
    return m


class _Signals:
    """The deterministic interference of one config, evaluated chunk by chunk on `device`."""

    def __init__(self, cfg: SKConfig, device):
        self.cfg, self.device = cfg, device
        two_pi = 2.0 * math.pi
        self.cw_f = [f for f in range(cfg.F) if cfg.cw_period and (f % cfg.cw_period) in cfg.cw_freqs]
        self.sine_f = [f for f in cfg.sine_freqs if f < cfg.F] if cfg.sine_inputs else []
        self.starts = burst_starts(cfg).tolist()
        f32 = torch.float32
        self.ph_blk = _phases(cfg, 1, (cfg.E,)).to(f32).to(device) if cfg.cw_block_inputs else None
        self.ph_cw = _phases(cfg, 2, (cfg.F, cfg.E)).to(f32).to(device) if self.cw_f else None
        self.ph_sine = _phases(cfg, 3, (cfg.F, cfg.E)).to(f32).to(device) if self.sine_f else None
        if self.starts:
            ph = _phases(cfg, 4, (cfg.F, cfg.E)).to(f32).to(device)
            self.burst_re = cfg.burst_amp * torch.cos(ph)
            self.burst_im = cfg.burst_amp * torch.sin(ph)
        self.two_pi = two_pi

    def _arg(self, nu: float, t64: torch.Tensor, ph: torch.Tensor) -> torch.Tensor:
        # 2 pi (nu t mod 1) in float64 keeps the phase accurate at large t; the rest is float32
        cyc = torch.remainder(nu * t64, 1.0).to(torch.float32)
        return self.two_pi * cyc[:, None] + ph[None, :]

    def chunk(self, t0: int, t1: int):
        """(re, im) float32 [t1-t0][F][E], or None if the chunk holds no interference."""
        cfg, device = self.cfg, self.device
        re = im = None

        def ensure():
            nonlocal re, im
            if re is None:
                re = torch.zeros(t1 - t0, cfg.F, cfg.E, dtype=torch.float32, device=device)
                im = torch.zeros_like(re)

        t64 = torch.arange(t0, t1, dtype=torch.float64, device=device)
        if cfg.cw_block_inputs is not None:
            blk, e0, ne = cfg.cw_block_inputs
            lo, hi = max(t0, blk * cfg.M), min(t1, (blk + 1) * cfg.M)
            if lo < hi:
                ensure()
                arg = self._arg(cfg.cw_cycles_per_sample, t64[lo - t0:hi - t0], self.ph_blk[e0:e0 + ne])
                re[lo - t0:hi - t0, 0, e0:e0 + ne] += cfg.cw_amp * torch.cos(arg)
                im[lo - t0:hi - t0, 0, e0:e0 + ne] += cfg.cw_amp * torch.sin(arg)
        for f in self.cw_f:
            ensure()
            nu = cfg.cw_cycles_per_sample * (1.0 + 0.01 * f)   # a slightly different tone per channel
            arg = self._arg(nu, t64, self.ph_cw[f])
            re[:, f, :] += cfg.cw_amp * torch.cos(arg)
            im[:, f, :] += cfg.cw_amp * torch.sin(arg)
        for f in self.sine_f:
            ensure()
            ne = cfg.sine_inputs
            arg = self._arg(cfg.sine_cycles_per_sample, t64, self.ph_sine[f][:ne])
            re[:, f, :ne] += cfg.sine_amp * torch.cos(arg)      # a real sinusoid: real component only
        for s in self.starts:
            lo, hi = max(t0, s), min(t1, s + cfg.burst_len)
            if lo < hi:
                ensure()
                # same time on all frequencies and inputs; constant modulus, phase per (f, e)
                re[lo - t0:hi - t0] += self.burst_re[None]
                im[lo - t0:hi - t0] += self.burst_im[None]
        return (re, im) if re is not None else None


def _chunk_rows(cfg: SKConfig, max_samples: int) -> int:
    rows = max(1, max_samples // (cfg.F * cfg.E))
    if rows >= cfg.M:
        rows -= rows % cfg.M
    return min(rows, cfg.T)


def quantise(re: torch.Tensor, im: torch.Tensor) -> torch.Tensor:
    """Round to nearest, clip to [-7, 7], offset by 8, pack (re nibble high, im nibble low)."""
    qr = torch.clamp(torch.round(re), -7, 7).to(torch.int16) + 8
    qi = torch.clamp(torch.round(im), -7, 7).to(torch.int16) + 8
    return ((qr << 4) | qi).to(torch.uint8)


def make_frame(cfg: SKConfig, device="cpu", frame: int = 0, out: Optional[torch.Tensor] = None,
               max_chunk_samples: int = 1 << 24) -> torch.Tensor:
    """uint8 [T][F][E] on `device`.  `frame` selects an independent noise realisation."""
    device = torch.device(device)
    if out is None:
        out = torch.empty(cfg.T, cfg.F, cfg.E, dtype=torch.uint8, device=device)
    assert out.shape == (cfg.T, cfg.F, cfg.E) and out.dtype == torch.uint8
    sig = sigma_per_input(cfg).to(torch.float32).to(device)
    rows = _chunk_rows(cfg, max_chunk_samples)
    g = torch.Generator(device=device)
    signals = _Signals(cfg, device)
    for ci, t0 in enumerate(range(0, cfg.T, rows)):
        t1 = min(cfg.T, t0 + rows)
        g.manual_seed((cfg.seed * 1000003 + frame * 65537 + ci) & 0x7FFFFFFFFFFF)
        shape = (t1 - t0, cfg.F, cfg.E)
        re = torch.randn(shape, generator=g, device=device, dtype=torch.float32) * sig
        im = torch.randn(shape, generator=g, device=device, dtype=torch.float32) * sig
        s = signals.chunk(t0, t1)
        if s is not None:
            re += s[0]
            im += s[1]
        out[t0:t1] = quantise(re, im)
    return out


def make_float_noise(cfg: SKConfig, frame: int = 0):
    """(re, im) float64 [T][F][E] on the CPU: the un-quantised noise of the same recipe, without
    interference.  Used for the float-input oracle's null-moment pins."""
    sig = sigma_per_input(cfg)
    g = _cpu_gen(cfg.seed * 1000003 + frame * 65537 + 999)
    shape = (cfg.T, cfg.F, cfg.E)
    re = torch.randn(shape, generator=g, dtype=torch.float64) * sig
    im = torch.randn(shape, generator=g, dtype=torch.float64) * sig
    return re, im


def random_bytes(T: int, F: int, E: int, seed: int, device="cpu") -> torch.Tensor:
    """Uniform random bytes (all 256 values, so nibble 0 = -8 occurs): an adversarial buffer."""
    g = torch.Generator(device="cpu")
    g.manual_seed(seed)
    return torch.randint(0, 256, (T, F, E), generator=g, dtype=torch.uint8).to(device)


def digitiser_thresholds(sigma) -> torch.Tensor:
    """Input model of the App. B simulation (Gaussian components rounded to the
    nearest level and bounded to [-7, 7]): for every receiver the 14 cumulative probabilities
    P(round-and-clip(N(0, sigma_e^2)) <= j - 7) = Phi((j - 6.5) / sigma_e), j = 0..13, scaled to
    32-bit thresholds.  uint32 [E][14] (stored as int64-safe numpy-compatible uint32 values).
    Both the oracle's and the CUDA path's samplers take this table as an input."""
    sig = torch.as_tensor(sigma, dtype=torch.float64).reshape(-1, 1)
    edges = (torch.arange(14, dtype=torch.float64) - 6.5).reshape(1, -1)
    cdf = torch.special.ndtr(edges / sig)
    thr = torch.clamp(torch.floor(cdf * 4294967296.0), 0, 4294967295.0)
    return thr.to(torch.int64).to(torch.uint32)
