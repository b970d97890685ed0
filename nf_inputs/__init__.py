"""Seeded synthetic inputs for the near-field direct sum (shared by tests, bench and smoke).

This module holds NONE of the method's arithmetic (no cells, no kernel, no forces): it only
draws particle positions.  It serves both the CUDA path and the oracle, which otherwise share
no code.  Every array is generated once per run and the same float32 bits are handed to both
sides, so parity never depends on re-generating.

The five configs are BASELINE.json's ``configs`` (all L = 1, R = 2, eps = L / (40 n_side), unit
masses, float32 positions in [0, L)).  They stand in for the paper's evolving LCDM particle
distribution at ~67 particles per cell (sec. 2.5; sec. 4.3), which is
not in this container: nearly uniform / displaced-lattice at early times (Table 6, z = 90.5) and
strongly clustered at late times (z = 0.105).  The recipes follow SURVEY.md sec. 8(d) and are
restated in DESIGN.md.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, replace

import torch

__all__ = ["NFConfig", "CONFIGS", "config", "generate", "scaled"]


@dataclass(frozen=True)
class NFConfig:
    name: str
    n_side: int            # N = n_side^3 particles
    cpd: int               # cells per dimension
    kind: str              # "uniform" | "zeldovich" | "halos" | "zeldovich+halos"
    seed: int
    L: float = 1.0
    R: int = 2
    zel_rms: float = 0.0   # 3-D rms displacement in lattice spacings
    halo_frac: float = 0.0  # fraction of particles placed in Plummer halos
    n_halos: int = 0
    halo_a_cells: float = 0.1   # Plummer scale radius in cell widths
    halo_sigma_ln: float = 1.5  # log-normal sigma of halo member counts

    @property
    def n(self) -> int:
        return self.n_side ** 3

    @property
    def eps(self) -> float:
        return self.L / (40.0 * self.n_side)

    def describe(self) -> str:
        return (f"{self.name}: N={self.n_side}^3 cpd={self.cpd} kind={self.kind} "
                f"ppc={self.n / self.cpd ** 3:.2f} eps={self.eps:.3e} seed={self.seed}")


CONFIGS = {
    1: NFConfig("config1_uniform_32", 32, 9, "uniform", 1001),
    2: NFConfig("config2_zeldovich_128", 128, 31, "zeldovich", 1002, zel_rms=0.2),
    3: NFConfig("config3_uniform_256", 256, 63, "uniform", 1003),
    4: NFConfig("config4_halos_512", 512, 125, "halos", 1004, halo_frac=0.5, n_halos=20000),
    5: NFConfig("config5_zeldovich_halos_1024", 1024, 251, "zeldovich+halos", 1005,
                zel_rms=0.5, halo_frac=0.3, n_halos=20000),
}


def config(idx: int) -> NFConfig:
    return CONFIGS[idx]


def scaled(idx: int, n_side: int, cpd: int | None = None, n_halos: int | None = None) -> NFConfig:
    """Same recipe as config ``idx`` at a smaller size (parity-test cases the oracle finishes in seconds).

    ``cpd`` defaults to the value that keeps the config's particles-per-cell; ``n_halos`` to the
    value that keeps the mean halo membership.
    """
    base = CONFIGS[idx]
    if cpd is None:
        cpd = max(2 * base.R + 1, round(base.cpd * n_side / base.n_side))
    if n_halos is None:
        n_halos = max(1, round(base.n_halos * (n_side / base.n_side) ** 3)) if base.n_halos else 0
    return replace(base, name=f"{base.name}@{n_side}", n_side=n_side, cpd=cpd, n_halos=n_halos)


# ----------------------------------------------------------------------------------------------
def _gen(seed: int, device) -> torch.Generator:
    g = torch.Generator(device=device)
    g.manual_seed(seed)
    return g


def _wrap_unit(x: torch.Tensor) -> torch.Tensor:
    """Map to [0, 1) in float32; values that round up to 1.0f go to 0."""
    x = x - torch.floor(x)
    x = x.to(torch.float32)
    x[x >= 1.0] = 0.0
    return x


def _uniform(n: int, g: torch.Generator, device) -> torch.Tensor:
    return torch.rand((n, 3), generator=g, device=device, dtype=torch.float32)


def _zeldovich(n_side: int, rms_spacings: float, g: torch.Generator, device) -> torch.Tensor:
    """Lattice q = (i + 0.5)/n_side plus displacements psi of a Gaussian field with P(k) ~ k^-2.

    delta_k = w_k / k (white noise w), psi_k = i k delta_k / k^2, the 3-D rms of psi is rescaled to
    ``rms_spacings`` lattice spacings.  Particle order is lattice order (x slowest, z fastest).
    """
    ns = n_side
    k1 = torch.fft.fftfreq(ns, d=1.0 / ns, device=device).to(torch.float32) * (2 * math.pi)
    kz1 = torch.fft.rfftfreq(ns, d=1.0 / ns, device=device).to(torch.float32) * (2 * math.pi)
    w = torch.randn((ns, ns, ns), generator=g, device=device, dtype=torch.float32)
    wk = torch.fft.rfftn(w)
    del w
    kx = k1.view(ns, 1, 1)
    ky = k1.view(1, ns, 1)
    kz = kz1.view(1, 1, ns // 2 + 1)
    k2 = kx * kx + ky * ky + kz * kz
    k2[0, 0, 0] = 1.0
    # psi_k = i k w_k / k^3 ; zero the DC mode and the Nyquist planes
    amp = wk * k2.pow(-1.5)
    del wk
    amp[0, 0, 0] = 0
    if ns % 2 == 0:
        amp[ns // 2, :, :] = 0
        amp[:, ns // 2, :] = 0
        amp[:, :, ns // 2] = 0
    psi = []
    for kk in (kx, ky, kz):
        comp = torch.fft.irfftn(1j * kk * amp, s=(ns, ns, ns))
        psi.append(comp.reshape(-1))
        del comp
    del amp, k2
    ms = sum((p.double() ** 2).mean().item() for p in psi)
    scale = (rms_spacings / ns) / math.sqrt(ms) if ms > 0 else 0.0
    q1 = (torch.arange(ns, device=device, dtype=torch.float32) + 0.5) / ns
    pos = torch.empty((ns ** 3, 3), device=device, dtype=torch.float32)
    for d, p in enumerate(psi):
        shape = [1, 1, 1]
        shape[d] = ns
        q = q1.view(shape).expand(ns, ns, ns).reshape(-1)
        pos[:, d] = _wrap_unit(q + p * scale)
    return pos


def _halo_members(m: int, cfg: NFConfig, g: torch.Generator, device, chunk: int = 1 << 25) -> torch.Tensor:
    """``m`` positions in ``cfg.n_halos`` Plummer spheres: centres uniform, member counts
    multinomial with log-normal weights (sigma_ln), scale radius a = halo_a_cells / cpd, radii
    truncated at 10 a (u <= 1.01^-1.5, equivalent to redrawing r > 10 a), isotropic directions."""
    nh = cfg.n_halos
    centres = torch.rand((nh, 3), generator=g, device=device, dtype=torch.float64)
    wts = torch.exp(cfg.halo_sigma_ln * torch.randn(nh, generator=g, device=device, dtype=torch.float64))
    cdf = torch.cumsum(wts, 0)
    cdf = cdf / cdf[-1]
    a = cfg.halo_a_cells / cfg.cpd
    umax = 1.01 ** -1.5
    out = torch.empty((m, 3), device=device, dtype=torch.float32)
    for s in range(0, m, chunk):
        e = min(m, s + chunk)
        k = e - s
        h = torch.searchsorted(cdf, torch.rand(k, generator=g, device=device, dtype=torch.float64))
        h.clamp_(max=nh - 1)
        u = torch.rand(k, generator=g, device=device, dtype=torch.float64) * umax
        u.clamp_(min=1e-12)
        r = a / torch.sqrt(u.pow(-2.0 / 3.0) - 1.0)
        v = torch.randn((k, 3), generator=g, device=device, dtype=torch.float64)
        v = v / v.norm(dim=1, keepdim=True).clamp_(min=1e-30)
        out[s:e] = _wrap_unit(centres[h] + v * r.unsqueeze(1))
    return out


def generate(cfg: NFConfig, device="cpu") -> torch.Tensor:
    """float32 positions [N][3] in [0, L), input order as described per kind."""
    device = torch.device(device)
    g = _gen(cfg.seed, device)
    n = cfg.n
    if cfg.kind == "uniform":
        pos = _uniform(n, g, device)
    elif cfg.kind == "zeldovich":
        pos = _zeldovich(cfg.n_side, cfg.zel_rms, g, device)
    elif cfg.kind == "halos":
        # halo members first (i < frac*n), then the uniform field particles
        m = int(round(cfg.halo_frac * n))
        pos = torch.empty((n, 3), device=device, dtype=torch.float32)
        pos[:m] = _halo_members(m, cfg, g, device)
        pos[m:] = _uniform(n - m, g, device)
    elif cfg.kind == "zeldovich+halos":
        pos = _zeldovich(cfg.n_side, cfg.zel_rms, g, device)
        moved = torch.rand(n, generator=g, device=device, dtype=torch.float32) < cfg.halo_frac
        idx = moved.nonzero(as_tuple=True)[0]
        del moved
        pos[idx] = _halo_members(idx.numel(), cfg, g, device)
    else:
        raise ValueError(cfg.kind)
    if cfg.L != 1.0:
        pos = pos * cfg.L
        pos[pos >= cfg.L] = 0.0
    return pos.contiguous()


def masses(cfg: NFConfig, device="cpu", sigma_ln: float = 1.0) -> torch.Tensor:
    """float32 masses [N] for the per-particle-mass variant (nf_set_masses): log-normal with median 1 (two decades of
    spread at sigma_ln = 1), seeded from the config; no arithmetic of the method in here."""
    device = torch.device(device)
    g = _gen(cfg.seed + 7919, device)
    return torch.exp(sigma_ln * torch.randn(cfg.n, generator=g, device=device, dtype=torch.float32)).contiguous()
