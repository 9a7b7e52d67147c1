"""Seeded synthetic inputs for the SHO project / add hot path.

This module holds NONE of the method's arithmetic (no Hermite functions, no boxes, no index maps):
it only draws atom positions, widths, wave functions and coefficients with the shapes, sizes and
value distributions of the five ``BASELINE.json`` configs (the paper's own workload, PAPER.md:369-371,
is measured on a synthetic crystal too; nothing here stands in for a public dataset).  It serves both
the CUDA path and the CPU oracle so that they see identical inputs; it imports neither.

Recipe: seed = 190500480 + k for config k.  Small arrays come from
``numpy.random.default_rng(seed)`` in the order positions -> sigma.  Large arrays are drawn per band
from ``default_rng([seed, 1000 + b])`` (psi) and per atom-block from ``default_rng([seed, 7])`` (coeff),
so that any band can be regenerated on its own; the HOST numpy array is the single source of truth.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

SEED0 = 190500480

_NP_DTYPE = {"r64": np.float64, "c128": np.complex128, "r32": np.float32, "c64": np.complex64}


@dataclass
class Workload:
    name: str
    seed: int
    ng: tuple            # (Nx, Ny, Nz)
    h: float             # grid spacing, Bohr
    periodic: tuple      # per axis 1/0
    kfrac: tuple | None  # Bloch phase per wrap = exp(2 pi i kfrac[d]); None for real data
    pos: np.ndarray      # [natoms][3], Bohr
    sigma: np.ndarray    # [natoms], Bohr
    numax: int
    nbands: int
    dtype: str           # "r64" | "c128" | "r32" | "c64"
    psi_dist: str        # "uniform" (U[-1,1]) | "normal" (N(0,1)) | "zero"
    rcut_sigma: float = 6.0
    note: str = ""
    extra: dict = field(default_factory=dict)

    @property
    def natoms(self) -> int:
        return int(self.pos.shape[0])

    @property
    def is_complex(self) -> bool:
        return self.dtype in ("c128", "c64")

    @property
    def np_dtype(self):
        return _NP_DTYPE[self.dtype]

    @property
    def npoints(self) -> int:
        return int(self.ng[0]) * int(self.ng[1]) * int(self.ng[2])

    def psi_band(self, b: int) -> np.ndarray:
        """Band b of psi, shape [Nz][Ny][Nx], in the workload's dtype (values drawn in fp64/fp32)."""
        shape = (self.ng[2], self.ng[1], self.ng[0])
        rng = np.random.default_rng([self.seed, 1000 + int(b)])
        real_t = np.float32 if self.dtype in ("r32", "c64") else np.float64

        def draw():
            if self.psi_dist == "uniform":
                return (rng.random(shape, dtype=real_t) * real_t(2) - real_t(1))
            if self.psi_dist == "normal":
                return rng.standard_normal(shape, dtype=real_t)
            if self.psi_dist == "zero":
                return np.zeros(shape, dtype=real_t)
            raise ValueError(self.psi_dist)

        if self.is_complex:
            out = np.empty(shape, dtype=self.np_dtype)
            out.real = draw()
            out.imag = draw()
            return out
        return draw()

    def psi(self, bands=None) -> np.ndarray:
        """psi[nb][Nz][Ny][Nx] (all bands, or the listed ones in the listed order)."""
        bands = range(self.nbands) if bands is None else bands
        return np.stack([self.psi_band(b) for b in bands], axis=0)

    def coeff(self, nsho: int) -> np.ndarray:
        """Coefficients c[natoms][nbands][nsho] ~ N(0,1) (re and im independent for complex)."""
        rng = np.random.default_rng([self.seed, 7])
        real_t = np.float32 if self.dtype in ("r32", "c64") else np.float64
        shape = (self.natoms, self.nbands, int(nsho))
        if self.is_complex:
            out = np.empty(shape, dtype=self.np_dtype)
            out.real = rng.standard_normal(shape, dtype=real_t)
            out.imag = rng.standard_normal(shape, dtype=real_t)
            return out
        return rng.standard_normal(shape, dtype=real_t)

    def dmatrix(self, nsho: int) -> np.ndarray:
        """Synthetic atomic matrices D[natoms][nsho][nsho] of step (2) (eq. (28) PAPER.md:252-262:
        real-valued, dimension N_SHO): fp64, symmetric, entries ~ N(0,1)/sqrt(nsho) (the real ones need PAW data)."""
        rng = np.random.default_rng([self.seed, 11])
        d = rng.standard_normal((self.natoms, int(nsho), int(nsho))) / np.sqrt(float(nsho))
        return np.ascontiguousarray(0.5 * (d + np.transpose(d, (0, 2, 1))))


def _lattice(rng, nsites, L, jitter):
    """Jittered simple-cubic sites (g + 1/2) L_d / n_d, z slowest, wrapped into the cell."""
    gx, gy, gz = np.meshgrid(np.arange(nsites[0]), np.arange(nsites[1]), np.arange(nsites[2]), indexing="ij")
    g = np.stack([gx, gy, gz], axis=-1).astype(np.float64)          # [nx][ny][nz][3]
    g = np.transpose(g, (2, 1, 0, 3)).reshape(-1, 3)                  # z slowest, x fastest
    site = (g + 0.5) * (np.asarray(L) / np.asarray(nsites, dtype=np.float64))
    p = site + rng.uniform(-jitter, jitter, size=site.shape)
    return np.mod(p, np.asarray(L))


def make(k: int, size: str = "full", dtype: str | None = None) -> Workload:
    """Config k (1..5) of BASELINE.json.  size="full" is the config as stated; size="small" keeps its
    structure (boundary type, box-to-cell ratio, overlap, numax, dtype) at a size the direct-sum oracle
    finishes in seconds.  ``dtype`` overrides the config's dtype (cfg 4 is stated for r32 and r64)."""
    seed = SEED0 + k
    rng = np.random.default_rng(seed)
    full = size == "full"
    if k == 1:
        # single atom at the cell centre (4,4,4) Bohr = grid point 16 (reading A2), isolated 32^3
        ng, h = (32, 32, 32), 0.25
        pos = np.array([[4.0, 4.0, 4.0]])
        sigma = np.array([1.0])
        return Workload("cfg1", seed, ng, h, (0, 0, 0), None, pos, sigma, 3, 1, dtype or "r64", "uniform",
                        note="single atom, isolated, box clipped to the grid")
    if k == 2:
        ng, h = ((96, 96, 96), 0.2) if full else ((48, 48, 48), 0.2)
        na, nb = (32, 16) if full else (6, 3)
        L = np.array(ng) * h
        pos = rng.uniform(0.0, 1.0, size=(na, 3)) * L
        sigma = rng.uniform(0.8, 1.2, size=na) if full else rng.uniform(0.5, 0.7, size=na)
        return Workload("cfg2" if full else "cfg2-small", seed, ng, h, (1, 1, 1), None, pos, sigma, 5, nb,
                        dtype or "r64", "normal", note="random atoms, sigma ~ U")
    if k == 3:
        ng, h = ((128, 128, 128), 0.2) if full else ((64, 64, 64), 0.2)
        sites, nb = ((8, 8, 4), 32) if full else ((4, 2, 2), 4)
        L = np.array(ng) * h
        pos = _lattice(rng, sites, L, 0.3)                      # reading A11: 8x8x4 sites
        sigma = np.full(pos.shape[0], 1.0 if full else 0.8)
        return Workload("cfg3" if full else "cfg3-small", seed, ng, h, (1, 1, 1), None, pos, sigma, 7, nb,
                        dtype or "r64", "normal", note="jittered lattice, on-the-fly vs stored tables")
    if k == 4:
        ng, h = ((128, 128, 128), 0.15) if full else ((48, 48, 48), 0.15)
        na, nb = (512, 32) if full else (12, 3)
        L = np.array(ng) * h
        pos = rng.uniform(0.0, 1.0, size=(na, 3)) * L
        sigma = np.full(na, 1.4 if full else 0.5)
        # reading A12: coefficients ~ N(0,1) are the input, psi_0 = 0
        return Workload("cfg4" if full else "cfg4-small", seed, ng, h, (1, 1, 1), None, pos, sigma, 7, nb,
                        dtype or "r64", "zero", note="add-back stress: heavily overlapping boxes")
    if k == 5:
        ng, h = ((192, 192, 192), 0.2) if full else ((48, 40, 56), 0.2)
        sites, nb = ((16, 8, 8), 64) if full else ((3, 2, 2), 3)
        L = np.array(ng) * h
        pos = _lattice(rng, sites, L, 0.3)                      # reading A11: 16x8x8 sites, jitter as cfg 3
        na = pos.shape[0]
        sigma = rng.uniform(0.7, 1.3, size=na) if full else rng.uniform(0.45, 0.6, size=na)
        return Workload("cfg5" if full else "cfg5-small", seed, ng, h, (1, 1, 1), (0.1, 0.2, 0.3), pos, sigma, 9,
                        nb, dtype or "c128", "normal", note="complex128 with Bloch phase")
    raise ValueError("config index must be 1..5")


BOHR_PER_ANGSTROM = 1.0 / 0.529177210903


def make_paper(numax: int = 5, dtype: str = "r64", size: str = "full") -> Workload:
    """The paper's own benchmark (sec. 6; tab. 1) as a second workload:
    an ISOLATED cubic domain of edge 16 Angstrom sampled with 64^3 points (h = 0.25 Angstrom), an fcc crystal
    with a = 4.08 Angstrom, every atom whose projection region of radius 3.55 Angstrom overlaps the domain
    (the paper counts 665), 1024 wave functions, 1 ... 56 projection coefficients (numax 0 ... 5), float and
    double.  Readings: a lattice point sits at the domain centre (that offset gives exactly
    665 atoms whose sphere overlaps the cube); the region is the CUBE |u_d| <= 3.55 Angstrom of reading A3, not
    the paper's sphere (1.9 times its volume); sigma = 3.55 Angstrom / 6 so that the configs' 6-sigma cut is that
    radius (the paper does not state sigma); everything in Bohr.  Nothing is drawn at random but psi.
    size="small": 24^3 points of the same spacing, 16 bands (for the parity tests)."""
    A = BOHR_PER_ANGSTROM
    full = size == "full"
    n = 64 if full else 24
    h = 0.25 * A
    L = n * 0.25                                     # Angstrom
    a, r = 4.08, 3.55
    basis = np.array([[0.0, 0.0, 0.0], [0.5, 0.5, 0.0], [0.5, 0.0, 0.5], [0.0, 0.5, 0.5]])
    rng_i = range(-8, 9)
    pts = np.array([(np.array([i, j, k]) + b) * a + 0.5 * L for i in rng_i for j in rng_i for k in rng_i for b in basis])
    d = np.maximum(np.maximum(-pts, pts - L), 0.0)
    keep = np.sqrt((d ** 2).sum(axis=1)) < r         # sphere of radius r overlaps the domain [0, L]^3
    pos = pts[keep]
    order = np.lexsort((pos[:, 0], pos[:, 1], pos[:, 2]))
    pos = np.ascontiguousarray(pos[order] * A)
    sigma = np.full(pos.shape[0], r * A / 6.0)
    nb = 1024 if full else 16
    return Workload("paper-nu%d" % numax if full else "paper-nu%d-small" % numax, SEED0 + 60 + numax, (n, n, n), h, (0, 0, 0),
                    None, pos, sigma, int(numax), nb, dtype, "normal",
                    note="paper sec. 6: isolated 16 A domain, fcc a = 4.08 A, r = 3.55 A, 1024 bands")
