"""Lattice builders with a fixed atom order (SURVEY.md §8d "Synthetic inputs").

Atom order: conventional-cell index ((ix*ny + iy)*nz + iz), basis atom fastest.
Cells are 3x3 row-major, rows = lattice vectors (h = (h1,h2,h3)^T).
"""
import numpy as np

FCC_BASIS = np.array([[0.0, 0.0, 0.0], [0.5, 0.5, 0.0], [0.5, 0.0, 0.5], [0.0, 0.5, 0.5]])
BCC_BASIS = np.array([[0.0, 0.0, 0.0], [0.5, 0.5, 0.5]])
DIAMOND_BASIS = np.concatenate([FCC_BASIS, FCC_BASIS + 0.25])


def _supercell(basis, nx, ny, nz, a):
    ix, iy, iz = np.meshgrid(np.arange(nx), np.arange(ny), np.arange(nz), indexing="ij")
    cells = np.stack([ix.ravel(), iy.ravel(), iz.ravel()], axis=1).astype(np.float64)  # (ncell,3)
    frac = (cells[:, None, :] + basis[None, :, :]).reshape(-1, 3)
    frac = frac / np.array([nx, ny, nz], dtype=np.float64)
    cell = np.diag([nx * a, ny * a, nz * a]).astype(np.float64)
    return frac, cell


def fcc_supercell(nx, ny, nz, a):
    """Fractional coordinates (n,3) and cell (3,3) of an nx x ny x nz conventional fcc supercell."""
    return _supercell(FCC_BASIS, nx, ny, nz, a)


def bcc_supercell(nx, ny, nz, a):
    """Fractional coordinates (n,3) and cell (3,3) of an nx x ny x nz conventional bcc supercell."""
    return _supercell(BCC_BASIS, nx, ny, nz, a)


def diamond_supercell(nx, ny, nz, a):
    """Fractional coordinates (n,3) and cell (3,3) of an nx x ny x nz conventional diamond-cubic supercell (8 atoms each)."""
    return _supercell(DIAMOND_BASIS, nx, ny, nz, a)


def bain_final_cell(cell_bcc, volume_ratio=1.0):
    """Bain-strained cell: c/a = sqrt(2) at constant volume (BASELINE.json configs[2]).

    Deformation diag(2^-1/6, 2^-1/6, 2^1/3) applied to the columns (x,y,z) of the
    bcc cell, then an isotropic scale volume_ratio^(1/3).
    """
    d = np.diag([2.0 ** (-1.0 / 6.0), 2.0 ** (-1.0 / 6.0), 2.0 ** (1.0 / 3.0)])
    return (cell_bcc @ d) * volume_ratio ** (1.0 / 3.0)
