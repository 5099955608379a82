"""Seeded synthetic inputs for the BASELINE.json configurations (C1..C5).

This module serves BOTH the CUDA path (tests, bench) and the CPU oracle with the *same* buffers.
It holds none of the method's arithmetic: no transforms of the solver, no eigenvalues, no
tridiagonal coefficients -- only grid spacings from the paper's closed-form stretching (eq. 7,
P:L236), random fields and a spectral *filter for generating inputs* (torch.fft, outside the
path under test).  The recipe is stated in DESIGN.md "Synthetic inputs"; the fields stand in for
the paper's turbulent-channel workload, whose data is not available.

Fields are torch float64 tensors of shape (nz, ny, nx), x fastest, generated on `device`
(CPU by default; the big configurations are generated on the GPU and copied to the host for the
oracle, so both sides always see identical bytes).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import Optional

import torch

SEED0 = 20010523400  # + config number (+10 * field index for u, v, w)


def tanh_grid(nz: int, lz: float, a: float):
    """Wall-normal grid clustered at both walls, eq. 7: z = lz/2 (1 + tanh(a(Z-1/2))/tanh(a/2)).

    Reading S10: the map is applied to the nz+1 *faces* Z_m = m/nz (so sum(dzf) = lz
    exactly); centres are face midpoints; dzc[k] is the distance between centres k-1 and k with
    mirror ghost centres outside both walls (dzc[0] = dzf[0], dzc[nz] = dzf[nz-1]).
    Returns (dzc[nz+1], dzf[nz], zc[nz]) as float64 CPU tensors.
    """
    Z = torch.arange(nz + 1, dtype=torch.float64) / nz
    zf = 0.5 * (1.0 + torch.tanh(a * (Z - 0.5)) / math.tanh(a * 0.5)) * lz
    zf[0] = 0.0
    zf[-1] = lz
    dzf = zf[1:] - zf[:-1]
    zc = 0.5 * (zf[1:] + zf[:-1])
    dzc = torch.empty(nz + 1, dtype=torch.float64)
    dzc[1:nz] = zc[1:] - zc[:-1]
    dzc[0] = dzf[0]
    dzc[nz] = dzf[nz - 1]
    return dzc, dzf, zc


def uniform_grid(nz: int, lz: float):
    h = lz / nz
    dzf = torch.full((nz,), h, dtype=torch.float64)
    dzc = torch.full((nz + 1,), h, dtype=torch.float64)
    zc = (torch.arange(nz, dtype=torch.float64) + 0.5) * h
    return dzc, dzf, zc


def _gen(seed: int, device) -> torch.Generator:
    g = torch.Generator(device=device)
    g.manual_seed(seed)
    return g


def uniform_field(shape, seed: int, device="cpu") -> torch.Tensor:
    """U[-1, 1] white noise."""
    g = _gen(seed, device)
    return torch.rand(shape, generator=g, dtype=torch.float64, device=device) * 2.0 - 1.0


def gaussian_field(shape, seed: int, device="cpu") -> torch.Tensor:
    g = _gen(seed, device)
    return torch.randn(shape, generator=g, dtype=torch.float64, device=device)


def kolmogorov_field(shape, lengths, seed: int, device="cpu") -> torch.Tensor:
    """White Gaussian noise filtered so that the shell-integrated spectrum goes like k^(-5/3):
    amplitude multiplied by |k|^(-11/6), |k| from the physical wavenumbers 2 pi m / L with the index
    space treated as periodic (for generation only), k = 0 zeroed, result scaled to unit RMS."""
    nz, ny, nx = shape
    lx, ly, lz = lengths
    x = gaussian_field(shape, seed, device)
    if torch.device(device).type == "cpu":
        # numpy's FFT on the host (torch's CPU irfftn aborted with heap corruption on the 16-core GPU box)
        import numpy as np
        xh = np.fft.rfftn(x.numpy())
        kx = 2.0 * math.pi * np.fft.rfftfreq(nx, d=lx / nx)
        ky = 2.0 * math.pi * np.fft.fftfreq(ny, d=ly / ny)
        kz = 2.0 * math.pi * np.fft.fftfreq(nz, d=lz / nz)
        k2 = kz[:, None, None] ** 2 + ky[None, :, None] ** 2 + kx[None, None, :] ** 2
        filt = np.where(k2 > 0, np.maximum(k2, 1e-300) ** (-11.0 / 12.0), 0.0)
        y = np.fft.irfftn(xh * filt, s=shape, axes=(0, 1, 2))
        y /= np.sqrt(np.mean(y * y))
        return torch.from_numpy(np.ascontiguousarray(y))
    xh = torch.fft.rfftn(x)
    del x
    kx = 2.0 * math.pi * torch.fft.rfftfreq(nx, d=lx / nx).to(device)
    ky = 2.0 * math.pi * torch.fft.fftfreq(ny, d=ly / ny).to(device)
    kz = 2.0 * math.pi * torch.fft.fftfreq(nz, d=lz / nz).to(device)
    k2 = kz[:, None, None] ** 2 + ky[None, :, None] ** 2 + kx[None, None, :] ** 2
    filt = torch.where(k2 > 0, k2.clamp_min(1e-300) ** (-11.0 / 12.0), torch.zeros_like(k2))
    del k2
    xh *= filt
    del filt
    y = torch.fft.irfftn(xh, s=shape)
    del xh
    y /= y.pow(2).mean().sqrt()
    return y.contiguous()


@dataclass
class Workload:
    name: str
    kind: str                       # "poisson" | "projection"
    n: tuple                        # (nx, ny, nz)
    lengths: tuple                  # (lx, ly, lz)
    bc: tuple                       # ((x_lo, x_up), (y_lo, y_up), (z_lo, z_up))
    dzc: Optional[torch.Tensor]     # CPU float64 (nz+1) or None (uniform)
    dzf: Optional[torch.Tensor]     # CPU float64 (nz)   or None (uniform)
    zc: torch.Tensor                # CPU float64 (nz) cell-centre heights
    dt: float = 1.0
    fields: dict = field(default_factory=dict)   # "f" or "u","v","w"

    @property
    def cells(self) -> int:
        return self.n[0] * self.n[1] * self.n[2]

    @property
    def bc_str(self) -> str:
        return "/".join(a + b for a, b in self.bc)


PI = math.pi

# name -> (kind, (nx,ny,nz), (lx,ly,lz), bc, stretching a or None)
CONFIGS = {
    "C1": ("poisson", (32, 32, 32), (2 * PI, PI, 2.0), (("P", "P"), ("P", "P"), ("N", "N")), None),
    "C2": ("poisson", (256, 128, 128), (2 * PI, PI, 2.0), (("P", "P"), ("P", "P"), ("N", "N")), 1.5),
    "C3": ("poisson", (512, 512, 256), (1.0, 1.0, 1.0), (("N", "N"), ("N", "N"), ("D", "N")), None),
    "C4": ("poisson", (1024, 512, 512), (4 * PI, 2.0, 2.0), (("P", "P"), ("D", "D"), ("N", "N")), 2.0),
    "C5": ("projection", (1024, 768, 512), (2 * PI, PI, 2.0), (("P", "P"), ("P", "P"), ("N", "N")), 1.6),
}
CONFIG_NUMBER = {"C1": 1, "C2": 2, "C3": 3, "C4": 4, "C5": 5}


def weighted_mean_removed(f: torch.Tensor, dzf: Optional[torch.Tensor]) -> torch.Tensor:
    """Subtract the dzf-weighted mean (volume mean) so that sum_k dzf_k sum_ij f = 0 (reading S3)."""
    if dzf is None:
        return f - f.mean()
    wz = (dzf / dzf.sum()).to(f.device)
    m = (f.mean(dim=(1, 2)) * wz).sum()
    return f - m


def make_workload(name: str, device="cpu", n_override=None, with_fields=True) -> Workload:
    """Build configuration `name` (C1..C5).  `n_override` = (nx, ny, nz) shrinks the grid while keeping
    the domain, boundary conditions, stretching and field recipe (used by tests and bounded CPU samples)."""
    kind, n, lengths, bc, a = CONFIGS[name]
    if n_override is not None:
        n = tuple(n_override)
    nx, ny, nz = n
    lx, ly, lz = lengths
    if a is None:
        dzc = dzf = None
        _, _, zc = uniform_grid(nz, lz)
    else:
        dzc, dzf, zc = tanh_grid(nz, lz, a)
    wl = Workload(name=name, kind=kind, n=n, lengths=lengths, bc=bc, dzc=dzc, dzf=dzf, zc=zc)
    if not with_fields:
        return wl
    shape = (nz, ny, nx)
    seed = SEED0 + CONFIG_NUMBER[name]
    if name == "C1":
        wl.fields["f"] = weighted_mean_removed(uniform_field(shape, seed, device), None)
    elif name == "C2":
        f = kolmogorov_field(shape, lengths, seed, device)
        wl.fields["f"] = weighted_mean_removed(f, dzf)
    elif name == "C3":
        wl.fields["f"] = uniform_field(shape, seed, device)
    elif name == "C4":
        # The 64-eigenmode part needs the operator's eigenvectors and is therefore assembled by the
        # tests from oracle tables; here only the 1e-3 Gaussian noise floor is generated.
        wl.fields["f"] = 1e-3 * gaussian_field(shape, seed, device)
    elif name == "C5":
        wl.dt = 1e-4
        zc_d = zc.to(device)
        prof = 6.0 * (zc_d / lz) * (1.0 - zc_d / lz)            # Poiseuille, bulk velocity 1
        for idx, comp in enumerate(("u", "v", "w")):
            g = kolmogorov_field(shape, lengths, seed + 10 * (idx + 1), device)
            g *= 0.1
            if comp == "u":
                g += prof[:, None, None]
            if comp == "w":
                g[nz - 1] = 0.0                                   # top wall; bottom wall face is implicit 0
            wl.fields[comp] = g
    return wl
