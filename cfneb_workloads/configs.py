"""BASELINE.json `configs` as seeded synthetic workloads.

Everything here is input preparation: lattice sites, linear interpolation in
(fractional coordinates, cell matrix) and additive seeded noise.  Potential
parameters are plain numbers copied from BASELINE.json; no potential is
evaluated here.
"""
import json
import os
from dataclasses import dataclass, field

import numpy as np

from .lattices import fcc_supercell, bcc_supercell, bain_final_cell, diamond_supercell
from .noise import splitmix64_normals

POT_LJ_SF = 0
POT_FS_MORSE = 1
POT_SW = 2
POT_DNN = 3
POT_NEP = 4


def lj_params(eps=1.0, sigma=1.0, rc=2.5):
    """Lennard-Jones shifted-force parameters: pot[0..2] = eps, sigma, r_c (BASELINE.json configs[0])."""
    p = np.zeros(12)
    p[0], p[1], p[2] = eps, sigma, rc
    return p


def sw_params(eps=2.1683, sigma=2.0951, a=1.80, lam=21.0, gamma=1.20, A=7.049556277, B=0.6022245584, p=4.0, q=0.0):
    """Stillinger-Weber parameters (the published silicon set: eV, Angstrom), padded to 12 doubles.

    Layout: eps, sigma, a (cut-off r_c = a sigma), lambda, gamma, A, B, p, q.  The functional form lives in the
    oracle and in the CUDA path separately; this is data only.
    """
    out = np.zeros(12)
    out[:9] = [eps, sigma, a, lam, gamma, A, B, p, q]
    return out


def dn_params(rc=4.2, K=4, M=3, L=3, H=8, seed=20251016):
    """Descriptor-network stand-in for the paper's NEP potential: cut-off, number of radial descriptors, angular
    radial functions, angular orders, hidden neurons, weight seed (layout of include/cfneb.h).  Data only."""
    out = np.zeros(12)
    out[:6] = [rc, K, M, L, H, seed]
    return out


def nep_params(rc_r=7.0, rc_a=4.6, n_r=6, n_a=4, k_r=8, k_a=8, L=4, H=32, n_types=2, seed=20251016):
    """NEP-shaped potential (the descriptor network widened to the shape of NEP proper): radial / angular cut-offs,
    radial descriptors, angular radial functions, basis sizes, Legendre orders, hidden neurons, atom types, weight
    seed (layout of include/cfneb.h).  Data only."""
    out = np.zeros(12)
    out[:10] = [rc_r, rc_a, n_r, n_a, k_r, k_a, L, H, n_types, seed]
    return out


def two_sublattice_types(n_atoms, n_types=2):
    """Atom types of the synthetic two-species crystal: zincblende ordering of the diamond generators' atom order
    (8 basis atoms per conventional cell, the first four on one fcc sublattice, the last four on the other)."""
    return (((np.arange(n_atoms) % 8) // 4) % max(int(n_types), 1)).astype(np.int32)


def diamond_strain_band(dims, a, n_images, seed, sigma_noise, strain, noise_endpoints=True):
    """A band of a diamond-cubic supercell between the cubic cell and the cell deformed by (I + strain), linear in the
    cell, fractional coordinates fixed, Gaussian noise on every image (on the endpoints too unless noise_endpoints is
    false) so that no atom sits on a symmetric site.  Returns pos[P,N,3], cells[P,3,3]."""
    frac, cell0 = diamond_supercell(dims[0], dims[1], dims[2], a)
    cell1 = cell0 @ (np.eye(3) + np.asarray(strain, dtype=np.float64))
    P, N = int(n_images), frac.shape[0]
    noise = splitmix64_normals(seed, P * N * 3).reshape(P, N, 3) * sigma_noise
    pos = np.empty((P, N, 3))
    cells = np.empty((P, 3, 3))
    for p in range(P):
        t = p / (P - 1)
        cells[p] = cell0 + t * (cell1 - cell0)
        pos[p] = frac @ cells[p] + (noise[p] if (noise_endpoints or 0 < p < P - 1) else 0.0)
    return pos, cells


def fs_params(D=0.3, alpha=1.5, r0=2.5, beta=3.0, rho_r0=2.5, A=0.8, r_on=4.5, r_cut=5.0):
    """Finnis-Sinclair-type parameters (BASELINE.json configs[2]).

    pot[0..7] = D, alpha, r0 (Morse pair), beta, rho_r0 (density exp(-beta (r - rho_r0))),
    A (embedding F = -A sqrt(rho)), r_on, r_cut (cosine taper).
    """
    p = np.zeros(12)
    p[:8] = [D, alpha, r0, beta, rho_r0, A, r_on, r_cut]
    return p


@dataclass
class WorkloadSpec:
    name: str
    potential: int
    pot: np.ndarray
    lattice: str  # "fcc_vacancy" | "bcc_bain" | "diamond_strain"
    dims: tuple
    n_atoms: int
    n_images: int
    seed: int
    noise_sigma: float = 1e-3
    k_spring: float = 1.0
    climb: bool = True
    n_steps: int = 200
    max_images: int = 0
    # FIRE (SURVEY.md §8c O7 defaults; dt's are per-config inputs)
    fire: dict = field(default_factory=dict)
    skin: float = 0.3
    max_neighbors: int = 128
    disorder_sigma: float = 0.0  # static Gaussian displacement of every atom, the same in all images (endpoints too)

    @property
    def types(self):
        """Atom types (NEP-shaped potential only; None otherwise)."""
        return two_sublattice_types(self.n_atoms, int(self.pot[8])) if self.potential == POT_NEP else None

    @property
    def r_cut(self):
        if self.potential == POT_NEP:
            return float(self.pot[0])
        if self.potential == POT_SW:
            return float(self.pot[2] * self.pot[1])
        if self.potential == POT_DNN:
            return float(self.pot[0])
        return float(self.pot[2] if self.potential == POT_LJ_SF else self.pot[7])


_FIRE_LJ = dict(dt0=0.01, dtmax=0.05, maxstep=0.1, nmin=5, finc=1.1, fdec=0.5, astart=0.1, fa=0.99)
_FIRE_EV = dict(dt0=0.1, dtmax=1.0, maxstep=0.2, nmin=5, finc=1.1, fdec=0.5, astart=0.1, fa=0.99)
_FIRE_SW = dict(dt0=0.02, dtmax=0.15, maxstep=0.05, nmin=5, finc=1.1, fdec=0.5, astart=0.1, fa=0.99)
_FIRE_DNN = dict(dt0=0.005, dtmax=0.02, maxstep=0.002, nmin=5, finc=1.1, fdec=0.5, astart=0.1, fa=0.99)
_FIRE_NEP = dict(dt0=0.005, dtmax=0.02, maxstep=0.002, nmin=5, finc=1.1, fdec=0.5, astart=0.1, fa=0.99)
_SW_STRAIN = ((0.0, 0.03, 0.0), (0.02, -0.03, 0.0), (0.0, 0.01, 0.04))

CONFIGS = [
    WorkloadSpec("c0_lj_vacancy_2x2x2", POT_LJ_SF, lj_params(), "fcc_vacancy", (2, 2, 2), 31, 7, 0,
                 fire=_FIRE_LJ, n_steps=200, max_images=7, skin=0.3, max_neighbors=128),
    WorkloadSpec("c1_lj_vacancy_4x4x4", POT_LJ_SF, lj_params(), "fcc_vacancy", (4, 4, 4), 255, 9, 1,
                 fire=_FIRE_LJ, n_steps=2000, max_images=9, skin=0.3, max_neighbors=128),
    WorkloadSpec("c2_fs_bain_2048", POT_FS_MORSE, fs_params(), "bcc_bain", (8, 8, 16), 2048, 16, 2,
                 fire=_FIRE_EV, n_steps=200, max_images=16, skin=0.3, max_neighbors=192),
    WorkloadSpec("c3_fs_bain_9826_adaptive", POT_FS_MORSE, fs_params(), "bcc_bain", (17, 17, 17), 9826, 12, 3,
                 fire=_FIRE_EV, n_steps=200, max_images=32, skin=0.3, max_neighbors=192),
    WorkloadSpec("c4_fs_bain_101306", POT_FS_MORSE, fs_params(), "bcc_bain", (37, 37, 37), 101306, 100, 4,
                 fire=_FIRE_EV, n_steps=500, max_images=100, skin=0.5, max_neighbors=224),
    # not a BASELINE.json config: the many-body (three-body) workload of SURVEY.md section 8(f) item 4, standing in for
    # the paper's NEP potential -- Stillinger-Weber diamond, 16^3 conventional cells x 32 images under a general strain
    WorkloadSpec("c5_sw_diamond_32768", POT_SW, sw_params(), "diamond_strain", (16, 16, 16), 32768, 32, 5,
                 noise_sigma=0.02, climb=False, fire=_FIRE_SW, n_steps=200, max_images=32, skin=0.3, max_neighbors=64),
    # the same band with the descriptor-network potential (the shape of NEP, seeded weights): 16 neighbours inside the
    # cut-off, 13 descriptors, 8 neurons.  The energy surface is arbitrary, so FIRE takes tiny steps: a cost workload
    WorkloadSpec("c6_dnn_diamond_32768", POT_DNN, dn_params(), "diamond_strain", (16, 16, 16), 32768, 32, 6,
                 noise_sigma=0.02, climb=False, fire=_FIRE_DNN, n_steps=100, max_images=32, skin=0.3, max_neighbors=64),
    # not a BASELINE.json config: configs[4] with every atom displaced by a static Gaussian kick of 0.12 A (the same in
    # all images, endpoints included) -- the paper's large bands are nucleated, locally disordered structures (P:18,
    # P:22), where the k-th neighbours of a warp's atoms no longer share a shell.  Throughput only.
    # Small FIRE steps: the kicked lattice is far from any minimum (forces of tens of eV/A, the endpoints included and
    # fixed), and the point is the cost of an iteration while the disorder is there, not where this band would end up.
    WorkloadSpec("c7_fs_bain_101306_disordered", POT_FS_MORSE, fs_params(), "bcc_bain", (37, 37, 37), 101306, 100, 4,
                 fire=dict(dt0=0.005, dtmax=0.02, maxstep=0.01, nmin=5, finc=1.1, fdec=0.5, astart=0.1, fa=0.99),
                 n_steps=500, max_images=100, skin=0.5, max_neighbors=224, disorder_sigma=0.12),
    # not a BASELINE.json config: the many-body workload at the shape and cost of NEP proper (SURVEY.md section 8(f)
    # item 4) -- the c5 band as a two-species (zincblende-ordered) crystal, 70 atoms inside the radial
    # cut-off of 7 A and 28 inside the angular one of 4.6 A, 6 + 4 x 4 = 22 descriptors, Legendre orders 1..4, 32 neurons
    # per type, type-pair expansion coefficients.  Seeded weights: cost and data flow, no physics.
    WorkloadSpec("c8_nep_diamond_32768", POT_NEP, nep_params(), "diamond_strain", (16, 16, 16), 32768, 32, 8,
                 noise_sigma=0.02, climb=False, fire=_FIRE_NEP, n_steps=100, max_images=32, skin=0.3, max_neighbors=128),
]


def load_lattice_constants():
    """Relaxed lattice constants written by `oracle/make_lattice_constants.py` (calls only oracle/).

    Keys: lj_fcc_a (sigma), fs_bcc_a (Angstrom), fs_fcc_volume_ratio (Omega_fcc / Omega_bcc per atom).
    """
    path = os.path.join(os.path.dirname(__file__), "lattice_constants.json")
    with open(path) as fh:
        return json.load(fh)


def vacancy_endpoints_unrelaxed(n, a):
    """fcc n^3 conventional cells minus atom 0; final = the atom at (1/2,1/2,0)a of cell 0 moved to the origin.

    Returns (frac_init, cell, frac_final, cell) with N = 4 n^3 - 1 atoms, unrelaxed.
    """
    frac, cell = fcc_supercell(n, n, n, a)
    frac_init = frac[1:].copy()  # remove atom 0 (origin site)
    frac_final = frac_init.copy()
    frac_final[0] = frac[0]  # former atom 1 = (1/2,1/2,0)a of cell 0 hops into the vacancy
    return frac_init, cell, frac_final, cell.copy()


def bain_endpoints(dims, a_bcc, volume_ratio=1.0):
    """bcc supercell and its Bain-strained (c/a = sqrt 2) image; fractional coordinates are identical."""
    frac, cell = bcc_supercell(dims[0], dims[1], dims[2], a_bcc)
    return frac, cell, frac.copy(), bain_final_cell(cell, volume_ratio)


def linear_path(frac0, cell0, frac1, cell1, n_images, seed, sigma):
    """Images linear in (fractional coordinates, cell matrix) + Gaussian noise on interior images.

    Returns Cartesian positions pos[P,N,3] = s_p h_p (+ noise, interior only) and cells[P,3,3].
    Positions are never wrapped.
    """
    P = int(n_images)
    N = frac0.shape[0]
    pos = np.empty((P, N, 3))
    cells = np.empty((P, 3, 3))
    noise = splitmix64_normals(seed, (P - 2) * N * 3).reshape(P - 2, N, 3) * sigma if P > 2 else None
    for p in range(P):
        t = p / (P - 1)
        s = frac0 + t * (frac1 - frac0)
        h = cell0 + t * (cell1 - cell0)
        pos[p] = s @ h
        cells[p] = h
        if 0 < p < P - 1:
            pos[p] += noise[p - 1]
    return pos, cells


def load_vacancy_endpoints(k):
    """Relaxed vacancy-hop endpoints of configs[k], k in (0, 1), written by `oracle/make_relaxed_endpoints.py`."""
    path = os.path.join(os.path.dirname(__file__), "vacancy_endpoints_c%d.json" % k)
    with open(path) as fh:
        d = json.load(fh)
    return (np.array(d["pos_init"]), np.array(d["cell_init"]), np.array(d["pos_final"]), np.array(d["cell_final"]))


def build_workload(k, n_images=None, dims=None):
    """Seeded inputs of BASELINE.json configs[k]: (spec, pos[P,N,3] Cartesian, cells[P,3,3]).

    n_images / dims (Bain configs only) override the config's band length / supercell: the same recipe at
    another size (used for bounded CPU-baseline samples and for parity cases between the configs).

    Vacancy configs: stored relaxed endpoints, 7 / 9 images linear in (fractional coordinates, cell) + noise.
    Bain configs: perfect bcc at the stress-free lattice constant and its c/a = sqrt(2) image at the stress-free
    volume (both exact cell-relaxed endpoints of a perfect crystal), linear in the cell matrix (= linear in the
    deformation gradient D, since h = h0 D) + noise on interior images.
    """
    spec = CONFIGS[k]
    P = int(n_images or spec.n_images)
    if spec.lattice == "fcc_vacancy":
        R0, h0, R1, h1 = load_vacancy_endpoints(k)
        pos, cells = linear_path(R0 @ np.linalg.inv(h0), h0, R1 @ np.linalg.inv(h1), h1, P, spec.seed, spec.noise_sigma)
    elif spec.lattice == "diamond_strain":
        pos, cells = diamond_strain_band(tuple(dims) if dims else spec.dims, 5.431, P, spec.seed, spec.noise_sigma, _SW_STRAIN,
                                         noise_endpoints=False)
    else:
        lc = load_lattice_constants()
        f0, c0, f1, c1 = bain_endpoints(tuple(dims) if dims else spec.dims, lc["fs_bcc_a"], lc["fs_fcc_volume_ratio"])
        pos, cells = linear_path(f0, c0, f1, c1, P, spec.seed, spec.noise_sigma)
        if spec.disorder_sigma > 0.0:
            kick = splitmix64_normals(spec.seed + 100, pos[0].size).reshape(pos[0].shape) * spec.disorder_sigma
            pos = pos + kick[None]
    return spec, pos, cells
