"""Pins for oracle/forcefield.c (O2 neighbours, O3 potentials / forces / virial).

Each test checks the oracle against something other than itself: textbook values, closed-form
lattice sums over crystallographic shells, finite differences of the energy (Eq. 3 / Eq. 5 of
PAPER.md), invariances, and an independent numpy brute force over periodic images.
"""
import itertools

import numpy as np
import pytest

from cfneb_workloads import bcc_supercell, diamond_supercell, dn_params, fcc_supercell, fs_params, lj_params, sw_params
from oracle import forcefield as ff

LJ, FS, SW, DNN = 0, 1, 2, 3


def energy(R, h, kind, pot, rc, cap=400, brute=True):
    nb = ff.neighbors(R, h, h, rc, cap, brute=brute)
    return ff.energy_force_virial(R, h, h, kind, pot, nb)


def random_triclinic(rng, scale):
    return scale * (np.eye(3) + 0.15 * rng.standard_normal((3, 3)))


# ---------- textbook points of the pair functions (dimer in a huge box) ----------

def dimer(r, kind, pot, rc):
    h = np.eye(3) * 50.0
    R = np.array([[10.0, 10.0, 10.0], [10.0 + r, 10.0, 10.0]])
    return energy(R, h, kind, pot, rc)


def test_lj_shifted_force_textbook_points():
    # Standard LJ facts: phi(sigma) = 0, minimum -eps at 2^(1/6) sigma, phi(2.5) = -0.016316891136 eps,
    # phi'(2.5) = 0.038999477 eps/sigma (the usual truncation constants of the rc = 2.5 sigma LJ fluid).
    pot = lj_params()
    phi_c = -0.016316891136
    dphi_c = 0.0389994774528
    assert abs(4 * (2.5 ** -12 - 2.5 ** -6) - phi_c) < 1e-12
    E, F, V = dimer(1.0, LJ, pot, 2.5)
    assert abs(E - (0.0 - phi_c - (1.0 - 2.5) * dphi_c)) < 1e-12
    rmin = 2.0 ** (1.0 / 6.0)
    E, F, V = dimer(rmin, LJ, pot, 2.5)
    assert abs(E - (-1.0 - phi_c - (rmin - 2.5) * dphi_c)) < 1e-12
    # at the LJ minimum phi' = 0, so the SF force on atom 0 due to atom 1 is -phi'(rc) r_hat: repelled by dphi_c
    assert abs(F[0, 0] - (-dphi_c)) < 1e-12 and abs(F[1, 0] - dphi_c) < 1e-12
    # energy and force vanish continuously at the cut-off
    E, F, V = dimer(2.5 - 1e-9, LJ, pot, 2.5)
    assert abs(E) < 1e-15 and np.abs(F).max() < 1e-8
    E, F, V = dimer(2.5 + 1e-9, LJ, pot, 2.5)
    assert E == 0.0 and np.abs(F).max() == 0.0


def test_fs_dimer_textbook_points():
    # Morse minimum: v(r0) = -D; density exp(0) = 1 per atom; E = v + 2 F(1) = -0.3 - 2*0.8 = -1.9 eV.
    pot = fs_params()
    E, F, V = dimer(2.5, FS, pot, 5.0)
    assert abs(E - (-1.9)) < 1e-14
    # at r0: v' = 0; force from embedding only: f = 2 F'(1) psi'(r0) = 2 (-0.4)(-3) = 2.4 eV/A, attractive
    assert abs(F[0, 0] - 2.4) < 1e-13 and abs(F[1, 0] + 2.4) < 1e-13
    # taper: zero beyond 5.0, continuous value and slope at both ends
    E, F, V = dimer(5.0 + 1e-9, FS, pot, 5.0)
    assert E == 0.0
    E, F, V = dimer(5.0 - 1e-7, FS, pot, 5.0)
    assert abs(E) < 1e-6
    Ea, Fa, _ = dimer(4.5 - 1e-7, FS, pot, 5.0)
    Eb, Fb, _ = dimer(4.5 + 1e-7, FS, pot, 5.0)
    assert abs(Ea - Eb) < 1e-6 and abs(Fa[0, 0] - Fb[0, 0]) < 1e-5


# ---------- closed-form lattice sums over crystallographic shells ----------

def test_lj_fcc_shell_sum():
    # fcc shells inside rc = 2.5 sigma at a = 1.55: n = 12, 6, 24, 12, 24 at d sqrt(1..5), d = a/sqrt 2 (78 neighbours)
    a = 1.55
    d = a / np.sqrt(2.0)
    shells = [(12, 1), (6, 2), (24, 3), (12, 4), (24, 5)]
    assert d * np.sqrt(5) < 2.5 < d * np.sqrt(6)
    phi = lambda r: 4 * (r ** -12 - r ** -6)
    dphi = lambda r: 4 * (-12 * r ** -13 + 6 * r ** -7)
    e_shell = 0.5 * sum(n * (phi(d * np.sqrt(k)) - phi(2.5) - (d * np.sqrt(k) - 2.5) * dphi(2.5)) for n, k in shells)
    frac, cell = fcc_supercell(2, 2, 2, a)  # box 3.1 < 2 rc: periodic self-images
    for brute in (True, False):
        nb = ff.neighbors(frac @ cell, cell, cell, 2.5, 128, brute=brute)
        assert np.all(nb[0] == 78)
        E, F, V = ff.energy_force_virial(frac @ cell, cell, cell, LJ, lj_params(), nb)
        assert abs(E / len(frac) - e_shell) < 1e-12
        assert np.abs(F).max() < 1e-12  # perfect Bravais lattice: zero force


def test_fs_bcc_shell_sum():
    # bcc shells inside 5.0 A at a = 2.87: 8, 6, 12, 24, 8 at a*(sqrt3/2, 1, sqrt2, sqrt11/2, sqrt3): 58 neighbours.
    # SURVEY.md §8c pins: rho = 10.4579, E = -4.96677 eV/atom.
    a = 2.87
    shells = [(8, np.sqrt(3) / 2), (6, 1.0), (12, np.sqrt(2)), (24, np.sqrt(11) / 2), (8, np.sqrt(3))]
    t = lambda r: 1.0 if r <= 4.5 else 0.5 * (1 + np.cos(np.pi * (r - 4.5) / 0.5))
    v = lambda r: 0.3 * (np.exp(-3.0 * (r - 2.5)) - 2 * np.exp(-1.5 * (r - 2.5))) * t(r)
    psi = lambda r: np.exp(-3.0 * (r - 2.5)) * t(r)
    rho = sum(n * psi(a * x) for n, x in shells)
    e = 0.5 * sum(n * v(a * x) for n, x in shells) - 0.8 * np.sqrt(rho)
    assert abs(rho - 10.4579) < 1e-4 and abs(e - (-4.96677)) < 1e-5
    frac, cell = bcc_supercell(2, 3, 4, a)
    for brute in (True, False):
        nb = ff.neighbors(frac @ cell, cell, cell, 5.0, 128, brute=brute)
        assert np.all(nb[0] == 58)
        E, F, V, Ui, rho_i = ff.energy_force_virial(frac @ cell, cell, cell, FS, fs_params(), nb, per_atom=True)
        assert np.allclose(rho_i, rho, rtol=0, atol=1e-12)
        assert np.allclose(Ui, e, rtol=0, atol=1e-12)
        assert abs(E / len(frac) - e) < 1e-12
        assert np.abs(F).max() < 1e-11
        assert np.allclose(V, V[0, 0] * np.eye(3), atol=1e-9)  # cubic symmetry: isotropic virial


def test_stillinger_weber_textbook_points():
    """The published silicon parametrisation has its two defining properties built in: the perfect diamond crystal at
    a = 5.431 A has cohesive energy -2 eps = -4.3366 eV per atom (four bonds per atom at the pair minimum of depth
    eps, every bond angle tetrahedral: cos theta = -1/3, so the three-body term vanishes), and that lattice is
    stress free.  A trimer with a non-tetrahedral angle isolates the three-body term."""
    pot = sw_params()
    eps, sig, rc = pot[0], pot[1], pot[2] * pot[1]
    frac, cell = diamond_supercell(2, 2, 2, 5.431)
    nb = ff.neighbors(frac @ cell, cell, cell, rc + 0.3, 64)
    E, F, V, Ui, _ = ff.energy_force_virial(frac @ cell, cell, cell, SW, pot, nb, per_atom=True)
    assert np.all(nb[0] == 16)                                   # 4 first + 12 second neighbours inside r_c + 0.3
    assert abs(E / len(frac) + 2.0 * eps) < 2e-4 * eps           # -2 eps to the precision of the published constants
    assert np.allclose(Ui, Ui[0], atol=1e-12) and np.abs(F).max() < 1e-11
    assert np.abs(V).max() < 2e-3 * len(frac) * eps              # stress free at the published lattice constant
    # pair term alone: dimer at the bond length d = a sqrt(3)/4 has energy -eps (value and minimum)
    d = 5.431 * np.sqrt(3.0) / 4.0
    e = lambda r: dimer(r, SW, pot, rc)[0]
    assert abs(e(d) + eps) < 1e-4 * eps
    assert e(d - 0.01) > e(d) < e(d + 0.01)
    assert e(rc - 1e-9) == pytest.approx(0.0, abs=1e-12) and e(rc + 0.1) == 0.0
    # trimer: centre at the origin, two neighbours at distance d under angle theta: E = 2 phi2(d) + lam eps (cos + 1/3)^2 g(d)^2
    for theta in (np.pi / 2, 2.0, np.arccos(-1.0 / 3.0)):
        h = np.eye(3) * 40.0
        R = np.array([[20.0, 20.0, 20.0], [20.0 + d, 20.0, 20.0], [20.0 + d * np.cos(theta), 20.0 + d * np.sin(theta), 20.0]])
        E3 = energy(R, h, SW, pot, rc)[0]
        d12 = np.linalg.norm(R[1] - R[2])
        pair = 2.0 * e(d) + (e(d12) if d12 < rc else 0.0)
        g = np.exp(pot[4] * sig / (d - rc))
        # the end atoms see only one neighbour inside r_c unless d12 < r_c (then their own triplets count as well)
        if d12 >= rc:
            assert abs(E3 - pair - pot[3] * eps * (np.cos(theta) + 1.0 / 3.0) ** 2 * g * g) < 1e-12


def splitmix64(seed, n):
    out, state, mask = [], seed, (1 << 64) - 1
    for _ in range(n):
        state = (state + 0x9E3779B97F4A7C15) & mask
        z = state
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & mask
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & mask
        out.append(z ^ (z >> 31))
    return out


def test_descriptor_network_energy_against_library_polynomials():
    """CFNEB_POT_DNN (include/cfneb.h; the shape of the paper's NEP).  The generator is pinned on the published
    SplitMix64 test vector (seed 1234567); the site energies of a small irregular cluster are then rebuilt from
    numpy's Chebyshev and Legendre routines, a dense matrix product and tanh -- none of the oracle's loops."""
    assert splitmix64(1234567, 3) == [6457827717110365317, 3203168211198807973, 9817491932198370423]
    from numpy.polynomial import chebyshev, legendre
    pot = dn_params(rc=3.0, K=4, M=3, L=3, H=8, seed=99)
    rc, K, M, L, H = pot[0], 4, 3, 3, 8
    D = K + M * L
    u = 2.0 * (np.array([z >> 11 for z in splitmix64(99, H * D + 2 * H)], dtype=np.float64) / 2.0 ** 53) - 1.0
    W0 = u[:H * D].reshape(H, D) * np.where(np.arange(D) < K, 0.3 / 8.0, 0.3 / 40.0)
    b0, W1 = 0.5 * u[H * D:H * D + H], u[H * D + H:]
    rng = np.random.default_rng(4)
    R = 20.0 + 1.6 * rng.standard_normal((7, 3))
    h = np.eye(3) * 40.0
    E, F, V, Ui, _ = ff.energy_force_virial(R, h, h, DNN, pot, ff.neighbors(R, h, h, rc, 16, brute=True), per_atom=True)
    expect = np.zeros(len(R))
    n_in = 0
    for i in range(len(R)):
        rv = np.array([R[j] - R[i] for j in range(len(R)) if j != i and np.linalg.norm(R[j] - R[i]) < rc])
        q = np.zeros(D)
        if len(rv):
            r = np.linalg.norm(rv, axis=1)
            n_in += len(r)
            fc = 0.5 * (1.0 + np.cos(np.pi * r / rc))
            x = 2.0 * (r / rc - 1.0) ** 2 - 1.0
            fk = np.array([0.5 * (chebyshev.chebval(x, np.eye(4)[k]) + 1.0) * fc for k in range(4)])  # [k, j]
            q[:K] = fk[:K].sum(axis=1)
            cosm = (rv @ rv.T) / np.outer(r, r)
            for n in range(M):
                for l in range(1, L + 1):
                    q[K + n * L + l - 1] = np.sum(np.outer(fk[n], fk[n]) * legendre.legval(cosm, np.eye(4)[l]))
        expect[i] = W1 @ np.tanh(W0 @ q - b0)
    assert n_in >= 10                                  # the cluster is not a set of isolated atoms
    assert np.allclose(Ui, expect, rtol=0, atol=1e-13)
    assert abs(E - expect.sum()) < 1e-12
    # an isolated atom has q = 0: U = -sum W1 tanh(b0)
    R1 = np.array([[5.0, 5.0, 5.0], [25.0, 25.0, 25.0]])
    assert abs(energy(R1, h, DNN, pot, rc)[0] - 2.0 * (W1 @ np.tanh(-b0))) < 1e-14


# ---------- finite differences: Eq. 5 (forces) and Eq. 3 (virial = -dU/d eps under h' = h(I+eps)) ----------

def perturbed(kind, rng):
    if kind == LJ:
        frac, cell = fcc_supercell(2, 2, 2, 1.58)
        frac = frac[1:]  # vacancy
        pot, rc = lj_params(), 2.5
        cell = cell @ (np.eye(3) + 0.03 * rng.standard_normal((3, 3)))
        R = frac @ cell + 0.05 * rng.standard_normal(frac.shape)
    elif kind == FS:
        frac, cell = bcc_supercell(2, 2, 3, 2.6)
        pot, rc = fs_params(), 5.0
        cell = cell @ (np.eye(3) + 0.03 * rng.standard_normal((3, 3)))
        R = frac @ cell + 0.08 * rng.standard_normal(frac.shape)
    elif kind == DNN:  # descriptor network on a compressed diamond lattice: about 16-28 neighbours inside the cut-off
        frac, cell = diamond_supercell(2, 2, 2, 5.2)
        frac = frac[1:]
        pot = dn_params()
        rc = pot[0]
        cell = cell @ (np.eye(3) + 0.03 * rng.standard_normal((3, 3)))
        R = frac @ cell + 0.15 * rng.standard_normal(frac.shape)
    else:  # Stillinger-Weber, compressed diamond so that some second neighbours are inside the cut-off too
        frac, cell = diamond_supercell(2, 2, 2, 5.2)
        frac = frac[1:]  # vacancy
        pot = sw_params()
        rc = pot[2] * pot[1]
        cell = cell @ (np.eye(3) + 0.03 * rng.standard_normal((3, 3)))
        R = frac @ cell + 0.15 * rng.standard_normal(frac.shape)
    return R, cell, pot, rc


@pytest.mark.parametrize("kind", [LJ, FS, SW, DNN])
def test_forces_match_finite_differences(kind):
    rng = np.random.default_rng(11 + kind)
    R, h, pot, rc = perturbed(kind, rng)
    E0, F, V = energy(R, h, kind, pot, rc)
    eps = 1e-5
    for i, m in [(0, 0), (3, 1), (7, 2), (len(R) - 1, 0)]:
        Rp, Rm = R.copy(), R.copy()
        Rp[i, m] += eps
        Rm[i, m] -= eps
        fd = -(energy(Rp, h, kind, pot, rc)[0] - energy(Rm, h, kind, pot, rc)[0]) / (2 * eps)
        assert abs(fd - F[i, m]) < 1e-7 * max(1.0, np.abs(F).max())
    assert np.abs(F.sum(axis=0)).max() < 1e-11 * len(R)  # sum F = 0 (f^ij = -f^ji)


@pytest.mark.parametrize("kind", [LJ, FS, SW, DNN])
def test_virial_matches_strain_derivative(kind):
    rng = np.random.default_rng(5 + kind)
    R, h, pot, rc = perturbed(kind, rng)
    s = R @ np.linalg.inv(h)
    E0, F, V = energy(R, h, kind, pot, rc)
    eps = 1e-5
    for m in range(3):
        for n in range(3):
            e = np.zeros((3, 3))
            e[m, n] = eps
            hp, hm = h @ (np.eye(3) + e), h @ (np.eye(3) - e)  # Eq. 2, s fixed
            fd = -(energy(s @ hp, hp, kind, pot, rc)[0] - energy(s @ hm, hm, kind, pot, rc)[0]) / (2 * eps)
            assert abs(fd - V[m, n]) < 2e-7 * np.abs(V).max()
    assert np.abs(V - V.T).max() < 1e-11 * np.abs(V).max()  # central forces: symmetric virial


def test_virial_sign_and_trace_zero_at_energy_minimum():
    # compressed solid => tr V > 0 (pressure-like); tr V = 0 where dE/da = 0
    def E_a(a):
        frac, cell = fcc_supercell(2, 2, 2, a)
        return energy(frac @ cell, cell, LJ, lj_params(), 2.5)

    assert np.trace(E_a(1.45)[2]) > 0 > np.trace(E_a(1.70)[2])
    lo, hi = 1.45, 1.70  # golden-section minimisation of E(a) alone
    g = (np.sqrt(5) - 1) / 2
    for _ in range(80):
        x1, x2 = hi - g * (hi - lo), lo + g * (hi - lo)
        if E_a(x1)[0] < E_a(x2)[0]:
            hi = x2
        else:
            lo = x1
    a_min = 0.5 * (lo + hi)
    E, F, V = E_a(a_min)
    assert abs(np.trace(V)) < 5e-5 * 32  # golden section on E resolves a to ~1e-8 => tr V ~ 1e-6 N
    assert 1.54 < a_min < 1.57


# ---------- invariances ----------

@pytest.mark.parametrize("kind", [LJ, FS, SW, DNN])
def test_rigid_rotation_and_translation_invariance(kind):
    rng = np.random.default_rng(3 + kind)
    R, h, pot, rc = perturbed(kind, rng)
    E0, F0, V0 = energy(R, h, kind, pot, rc)
    Q, _ = np.linalg.qr(rng.standard_normal((3, 3)))
    E1, F1, V1 = energy(R @ Q, h @ Q, kind, pot, rc)
    assert abs(E1 - E0) < 1e-11 * abs(E0)
    assert np.abs(F1 - F0 @ Q).max() < 1e-11 * np.abs(F0).max()
    assert np.abs(V1 - Q.T @ V0 @ Q).max() < 1e-11 * np.abs(V0).max()
    shift = np.array([0.37, -1.2, 5.1])  # translation, including across the periodic boundary
    E2, F2, V2 = energy(R + shift, h, kind, pot, rc)
    assert abs(E2 - E0) < 1e-11 * abs(E0) and np.abs(F2 - F0).max() < 1e-10 * np.abs(F0).max()


# ---------- neighbours: independent numpy brute force, cell list vs brute force, symmetry ----------

def numpy_neighbors(R, h, r_list, reach=4):
    s = R @ np.linalg.inv(h)
    out = set()
    for n in itertools.product(range(-reach, reach + 1), repeat=3):
        d = (s[None, :, :] - s[:, None, :] + np.array(n, dtype=float)) @ h
        r2 = np.sum(d * d, axis=2)
        for i, j in zip(*np.nonzero(r2 < r_list * r_list)):
            if i == j and n == (0, 0, 0):
                continue
            out.add((int(i), int(j)) + n)
    return out


def as_set(nb):
    count, lst, shift = nb
    out = set()
    for i in range(len(count)):
        for k in range(count[i]):
            out.add((i, int(lst[i, k])) + tuple(int(x) for x in shift[i, k]))
    assert len(out) == int(count.sum())  # no duplicates
    return out


def test_neighbors_small_box_against_numpy_brute_force():
    # configs[0] geometry: box edge 2a = 3.1 sigma < 2 r_list: several periodic images of the same atom, self-images
    rng = np.random.default_rng(0)
    frac, cell = fcc_supercell(2, 2, 2, 1.557)
    R = (frac @ cell)[1:] + 0.05 * rng.standard_normal((31, 3)) + np.array([0.3, -0.2, 4.0])  # unwrapped, shifted
    for r_list in (2.8, 3.3):  # 3.3 > box edge: an atom is its own neighbour through the boundary
        ref = numpy_neighbors(R, cell, r_list)
        assert any(i == j for i, j, *_ in ref) == (r_list > 3.2)
        assert len({(i, j) for i, j, *_ in ref}) < len(ref)  # several images of the same neighbour
        for brute in (True, False):
            got = as_set(ff.neighbors(R, cell, cell, r_list, 400, brute=brute))
            assert got == ref
    assert all((j, i, -a, -b, -c) in ref for (i, j, a, b, c) in ref)  # (i;j,n) <=> (j;i,-n)


@pytest.mark.parametrize("seed", [1, 2, 3])
def test_cell_list_equals_brute_force_on_random_triclinic(seed):
    rng = np.random.default_rng(seed)
    n = 150
    h = random_triclinic(rng, [6.0, 9.0, 14.0][seed - 1])
    R = rng.uniform(-0.5, 1.5, (n, 3)) @ h  # unwrapped
    r_list = 2.2
    a = as_set(ff.neighbors(R, h, h, r_list, 400, brute=True))
    b = as_set(ff.neighbors(R, h, h, r_list, 400, brute=False))
    assert a == b
    if seed == 1:
        assert a == numpy_neighbors(R, h, r_list, reach=3)


def test_neighbors_use_image_cell_not_reference_cell():
    # Rt = s h0 is stored; distances are measured in the image's own cell h = h0 D (Eq. 10)
    rng = np.random.default_rng(4)
    frac, h0 = bcc_supercell(3, 3, 3, 2.3)
    D = np.eye(3) + 0.1 * rng.standard_normal((3, 3))
    h = h0 @ D
    Rt = frac @ h0 + 0.05 * rng.standard_normal(frac.shape)
    got = as_set(ff.neighbors(Rt, h0, h, 4.0, 300, brute=False))
    assert got == as_set(ff.neighbors(Rt, h0, h, 4.0, 300, brute=True))
    assert got == numpy_neighbors(Rt @ D, h, 4.0, reach=2)


def test_neighbor_overflow_is_an_error():
    frac, cell = fcc_supercell(2, 2, 2, 1.55)
    with pytest.raises(ff.OracleError) as e:
        ff.neighbors(frac @ cell, cell, cell, 2.5, 16)
    assert e.value.code == -4
