"""Seeded synthetic inputs shaped like the paper's workloads (BASELINE.json:configs).

This module serves BOTH the CUDA path and the oracle and therefore holds none of the
method's arithmetic: it only draws phantoms (refractive-index volumes), analytic input
beams and emitter lists.  It imports neither ``oracle`` nor the CUDA binding.

The paper's own samples (embryo phantom n = 1.33-1.38; embryo model
n = 1.35-1.39, line 27; grids of 1024^3 voxels, line 21) are not available; the five
configurations below stand in for them.  Recipe (restated in DESIGN.md "Inputs"):

* cell parameters come from ``numpy.random.default_rng(170602261 + c)`` (PCG64) for
  config c, drawn as whole arrays in the order centres[n][3] ~ U(0, L), radii, values;
* voxel i sits at coordinate i*dx; a voxel is inside a cell if its centre satisfies the
  ellipsoid inequality <= 1; cells are painted in index order, later ones overwrite
  earlier ones; no periodic wrap;
* smoothed noise: ``torch.randn`` (generator seeded with the same seed, on the device the
  volume is built on -- CPU and CUDA streams differ, so an array is generated ONCE and the
  same array is handed to both sides), blurred with a periodic separable Gaussian of
  sigma = 1 um, rescaled to standard deviation 0.005 and added after the cells;
* field pixel i sits at (i - N/2)*dx.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Optional, Tuple

import numpy as np
import torch

SEED_BASE = 170602261


@dataclasses.dataclass(frozen=True)
class Workload:
    name: str
    index: int                 # position in BASELINE.json:configs
    Nx: int
    Ny: int
    Nz: int
    dx: float                  # um
    dz: float                  # um
    lam: float                 # vacuum wavelength, um
    n0: float
    batch: int = 1
    field: str = "gaussian"    # gaussian | sheet | multiplex | gaussian_batch
    w0: float = 2.0            # um (gaussian)
    NA: float = 0.0            # sheet / multiplex
    emitters: int = 0          # per side of the emitter grid
    spacing: float = 0.0       # um
    n_cells: int = 0
    cell_shape: str = "sphere"  # sphere | ellipsoid
    r_lo: float = 2.0
    r_hi: float = 5.0
    dn_lo: float = 0.01
    dn_hi: float = 0.05
    noise_sigma_um: float = 0.0
    noise_amp: float = 0.0
    nref_slab: int = 32

    @property
    def seed(self) -> int:
        return SEED_BASE + self.index

    def with_nz(self, Nz: int) -> "Workload":
        """Same lateral problem, first ``Nz`` slices only (for bounded CPU samples)."""
        return dataclasses.replace(self, Nz=int(Nz))


CONFIGS = {
    # BASELINE.json:configs[0]
    "C1": Workload("C1", 0, 128, 128, 128, 0.1, 0.1, 0.5, 1.33, field="gaussian", w0=2.0,
                   n_cells=20, cell_shape="sphere", r_lo=2.0, r_hi=5.0, dn_lo=0.01, dn_hi=0.05),
    # configs[1]
    "C2": Workload("C2", 1, 256, 256, 256, 0.2, 0.2, 0.488, 1.33, field="sheet", NA=0.1,
                   n_cells=200, cell_shape="ellipsoid", r_lo=3.0, r_hi=8.0, dn_lo=0.01, dn_hi=0.04,
                   noise_sigma_um=1.0, noise_amp=0.005),
    # configs[2]
    "C3": Workload("C3", 2, 512, 512, 512, 0.2, 0.2, 0.5, 1.33, field="multiplex", NA=0.8,
                   emitters=10, spacing=8.0,
                   n_cells=1600, cell_shape="ellipsoid", r_lo=3.0, r_hi=8.0, dn_lo=0.01, dn_hi=0.04,
                   noise_sigma_um=1.0, noise_amp=0.005),
    # configs[3] -- the headline workload (~1000 PSFs through 1024^3 voxels)
    "C4": Workload("C4", 3, 1024, 1024, 1024, 0.1, 0.1, 0.5, 1.33, field="multiplex", NA=0.8,
                   emitters=32, spacing=3.2,
                   n_cells=2000, cell_shape="sphere", r_lo=2.0, r_hi=6.0, dn_lo=0.01, dn_hi=0.05,
                   noise_sigma_um=1.0, noise_amp=0.005),
    # configs[4]
    "C5": Workload("C5", 4, 512, 512, 512, 0.2, 0.2, 0.5, 1.33, batch=16, field="gaussian_batch",
                   n_cells=1600, cell_shape="ellipsoid", r_lo=3.0, r_hi=8.0, dn_lo=0.01, dn_hi=0.04,
                   noise_sigma_um=1.0, noise_amp=0.005),
}


def config(name: str) -> Workload:
    return CONFIGS[name]


def tiny(name: str = "T", N: int = 32, Nz: int = 8, **kw) -> Workload:
    """A small workload for brute-force checks (not one of the paper-shaped configs)."""
    base = dict(name=name, index=99, Nx=N, Ny=N, Nz=Nz, dx=0.2, dz=0.2, lam=0.5, n0=1.33,
                field="gaussian", w0=1.0, n_cells=6, cell_shape="ellipsoid",
                r_lo=0.5, r_hi=2.0, dn_lo=0.01, dn_hi=0.05)
    base.update(kw)
    return Workload(**base)


# ----------------------------------------------------------------------------------------
# refractive-index volumes
# ----------------------------------------------------------------------------------------
def _cell_params(w: Workload, rng: np.random.Generator):
    Lx, Ly, Lz = w.Nx * w.dx, w.Ny * w.dx, w.Nz * w.dz
    n = w.n_cells
    centres = rng.uniform(0.0, 1.0, size=(n, 3)) * np.array([Lx, Ly, Lz])
    if w.cell_shape == "sphere":
        r = rng.uniform(w.r_lo, w.r_hi, size=(n, 1))
        radii = np.repeat(r, 3, axis=1)
    else:
        radii = rng.uniform(w.r_lo, w.r_hi, size=(n, 3))
    vals = rng.uniform(w.dn_lo, w.dn_hi, size=(n,))
    return centres, radii, vals


def _periodic_gaussian_blur_(vol: torch.Tensor, sigmas_vox) -> torch.Tensor:
    """Separable periodic Gaussian blur along each axis of a 3-D float32 tensor."""
    for axis, sig in enumerate(sigmas_vox):
        if sig <= 0:
            continue
        n = vol.shape[axis]
        rad = int(min(math.ceil(4.0 * sig), (n - 1) // 2))
        t = torch.arange(-rad, rad + 1, dtype=torch.float64)
        k = torch.exp(-0.5 * (t / sig) ** 2)
        k = (k / k.sum()).to(torch.float32).to(vol.device)
        v = vol.movedim(axis, -1)
        shp = v.shape
        # chunk the leading dimension to bound the padded temporary
        rows = v.reshape(-1, 1, n)
        out = torch.empty_like(rows)
        step = max(1, (1 << 26) // n)
        for s in range(0, rows.shape[0], step):
            blk = rows[s:s + step]
            blk = torch.nn.functional.pad(blk, (rad, rad), mode="circular")
            out[s:s + step] = torch.nn.functional.conv1d(blk, k.view(1, 1, -1))
        vol = out.reshape(shp).movedim(-1, axis).contiguous()
    return vol


def make_dn(w: Workload, device="cpu") -> torch.Tensor:
    """float32 [Nz][Ny][Nx] volume of n - n0 (x fastest)."""
    dev = torch.device(device)
    rng = np.random.default_rng(w.seed)
    centres, radii, vals = _cell_params(w, rng)
    vol = torch.zeros((w.Nz, w.Ny, w.Nx), dtype=torch.float32, device=dev)
    xs = torch.arange(w.Nx, dtype=torch.float64, device=dev) * w.dx
    ys = torch.arange(w.Ny, dtype=torch.float64, device=dev) * w.dx
    zs = torch.arange(w.Nz, dtype=torch.float64, device=dev) * w.dz
    for (cx, cy, cz), (rx, ry, rz), v in zip(centres, radii, vals):
        x0, x1 = max(0, int(math.floor((cx - rx) / w.dx))), min(w.Nx, int(math.ceil((cx + rx) / w.dx)) + 1)
        y0, y1 = max(0, int(math.floor((cy - ry) / w.dx))), min(w.Ny, int(math.ceil((cy + ry) / w.dx)) + 1)
        z0, z1 = max(0, int(math.floor((cz - rz) / w.dz))), min(w.Nz, int(math.ceil((cz + rz) / w.dz)) + 1)
        if x0 >= x1 or y0 >= y1 or z0 >= z1:
            continue
        ex = ((xs[x0:x1] - cx) / rx) ** 2
        ey = ((ys[y0:y1] - cy) / ry) ** 2
        ez = ((zs[z0:z1] - cz) / rz) ** 2
        inside = (ez[:, None, None] + ey[None, :, None] + ex[None, None, :]) <= 1.0
        sub = vol[z0:z1, y0:y1, x0:x1]
        sub[inside] = float(v)
    if w.noise_amp > 0.0:
        gen = torch.Generator(device=dev)
        gen.manual_seed(w.seed)
        noise = torch.randn((w.Nz, w.Ny, w.Nx), dtype=torch.float32, device=dev, generator=gen)
        noise = _periodic_gaussian_blur_(noise, (w.noise_sigma_um / w.dz,
                                                 w.noise_sigma_um / w.dx,
                                                 w.noise_sigma_um / w.dx))
        std = float(noise.double().std())
        if std > 0:
            noise *= (w.noise_amp / std)
        vol += noise
        del noise
    return vol


# ----------------------------------------------------------------------------------------
# input fields (analytic shapes only; multiplexed fields are built by Algorithm M on the
# side under test, from the emitter lists below)
# ----------------------------------------------------------------------------------------
def _coords(N: int, dx: float) -> np.ndarray:
    return (np.arange(N, dtype=np.float64) - N // 2) * dx


def gaussian_beam(Nx: int, Ny: int, dx: float, w0: float, cx: float = 0.0, cy: float = 0.0) -> np.ndarray:
    """exp(-r^2 / w0^2), flat phase, waist at the input plane; complex64 [Ny][Nx]."""
    x = _coords(Nx, dx) - cx
    y = _coords(Ny, dx) - cy
    g = np.exp(-(y[:, None] ** 2 + x[None, :] ** 2) / (w0 * w0))
    return g.astype(np.complex64)


def light_sheet(Nx: int, Ny: int, dx: float, lam: float, n0: float, NA: float, z_focus: float) -> np.ndarray:
    """Cylindrically focused Gaussian sheet, flat in x, converging in y to a waist
    w0 = lam / (pi NA) at depth ``z_focus``: the paraxial 1-D Gaussian-beam profile at
    z = -z_focus, g(y) = q^{-1/2} exp(-y^2 / (w0^2 q)), q = 1 - i z_focus / zR,
    zR = pi w0^2 n0 / lam.  complex64 [Ny][Nx]."""
    w0 = lam / (math.pi * NA)
    zR = math.pi * w0 * w0 * n0 / lam
    q = 1.0 - 1j * z_focus / zR
    y = _coords(Ny, dx)
    g = np.exp(-(y ** 2) / (w0 * w0 * q)) / np.sqrt(q)
    return np.repeat(g[:, None], Nx, axis=1).astype(np.complex64)


def make_emitters(w: Workload) -> Tuple[np.ndarray, np.ndarray, np.ndarray]:
    """Emitter grid of a multiplex workload: pos float32 [M][2] (x, y) in um relative to the
    centre pixel, phase float32 [M] ~ U(0, 2 pi), amp float32 [M] = 1."""
    assert w.field == "multiplex"
    rng = np.random.default_rng(w.seed + 1000)
    m = w.emitters
    g = (np.arange(m, dtype=np.float64) - (m - 1) / 2.0) * w.spacing
    px, py = np.meshgrid(g, g, indexing="xy")
    pos = np.stack([px.ravel(), py.ravel()], axis=1).astype(np.float32)
    phase = rng.uniform(0.0, 2.0 * math.pi, size=(m * m,)).astype(np.float32)
    amp = np.ones((m * m,), dtype=np.float32)
    return pos, phase, amp


def make_field(w: Workload) -> Optional[np.ndarray]:
    """complex64 [B][Ny][Nx] for analytic input fields; ``None`` for multiplex workloads
    (their field is Algorithm M applied to :func:`make_emitters`)."""
    if w.field == "gaussian":
        return gaussian_beam(w.Nx, w.Ny, w.dx, w.w0)[None]
    if w.field == "sheet":
        return light_sheet(w.Nx, w.Ny, w.dx, w.lam, w.n0, w.NA, 0.5 * w.Nz * w.dz)[None]
    if w.field == "gaussian_batch":
        rng = np.random.default_rng(w.seed + 2000)
        L = w.Nx * w.dx
        w0s = rng.uniform(1.0, 3.0, size=(w.batch,))
        off = rng.uniform(-L / 4.0, L / 4.0, size=(w.batch, 2))
        return np.stack([gaussian_beam(w.Nx, w.Ny, w.dx, w0s[b], off[b, 0], off[b, 1])
                         for b in range(w.batch)])
    if w.field == "multiplex":
        return None
    raise ValueError(w.field)


def random_field(Nx: int, Ny: int, seed: int, batch: int = 1) -> np.ndarray:
    """Seeded complex Gaussian noise, complex64 [B][Ny][Nx] (FFT / kernel unit tests)."""
    rng = np.random.default_rng(seed)
    a = rng.standard_normal((batch, Ny, Nx)) + 1j * rng.standard_normal((batch, Ny, Nx))
    return a.astype(np.complex64)
