"""Pins for oracle/cellfilter.py: Eq. 10-17 of PAPER.md checked by finite differences of the energy,
by rotation invariance and by the defining properties of the matrix square root."""
import numpy as np
import pytest

from cfneb_workloads import bcc_supercell, fcc_supercell, fs_params, lj_params
from oracle import cellfilter as cf
from oracle import forcefield as ff


def system(kind, rng):
    if kind == 0:
        frac, h0 = fcc_supercell(2, 2, 2, 1.58)
        pot, rc = lj_params(), 2.5
    else:
        frac, h0 = bcc_supercell(2, 2, 3, 2.6)
        pot, rc = fs_params(), 5.0
    h0 = h0 @ (np.eye(3) + 0.02 * rng.standard_normal((3, 3)))
    D = np.eye(3) + 0.06 * rng.standard_normal((3, 3))  # general (non-symmetric) deformation gradient
    Rt = frac @ h0 + 0.05 * rng.standard_normal(frac.shape)
    return Rt, h0, D, pot, rc


def E_of(Rt, h0, D, kind, pot, rc):
    """Energy as a function of the paper's variables (R~, D): R = R~ D, h = h0 D (Eq. 10)."""
    h = h0 @ D
    nb = ff.neighbors(Rt, h0, h, rc, 400, brute=True)
    return ff.energy_force_virial(Rt, h0, h, kind, pot, nb)


@pytest.mark.parametrize("kind", [0, 1])
def test_input_mapping_eq10_eq15(kind):
    rng = np.random.default_rng(kind)
    Rt, h0, D, pot, rc = system(kind, rng)
    R, h = Rt @ D, h0 @ D
    Rt2, B, D2 = cf.input_mapping(R, h, h0)
    assert np.allclose(D2, D, atol=1e-13) and np.allclose(B, D @ D.T, atol=1e-13)
    assert np.allclose(Rt2, Rt, atol=1e-12)
    s = R @ np.linalg.inv(h)
    assert np.allclose(Rt2, s @ h0, atol=1e-12)  # R~ = s h0 (Eq. 10)


@pytest.mark.parametrize("kind", [0, 1])
def test_atomic_generalized_force_eq12(kind):
    # -dE/dR~ at fixed D equals F D^T
    rng = np.random.default_rng(10 + kind)
    Rt, h0, D, pot, rc = system(kind, rng)
    E, F, V = E_of(Rt, h0, D, kind, pot, rc)
    G = cf.generalized_force(F, V, D, 1.0, cf.CELL_D)
    eps = 1e-5
    for i, m in [(0, 0), (2, 1), (5, 2)]:
        Rp, Rm = Rt.copy(), Rt.copy()
        Rp[i, m] += eps
        Rm[i, m] -= eps
        fd = -(E_of(Rp, h0, D, kind, pot, rc)[0] - E_of(Rm, h0, D, kind, pot, rc)[0]) / (2 * eps)
        assert abs(fd - G[i, m]) < 1e-7 * np.abs(G[:-3]).max()
    assert not np.allclose(G[:-3], F, atol=1e-3)  # D^T matters


@pytest.mark.parametrize("kind", [0, 1])
def test_cell_generalized_force_eq13_eq14(kind):
    # -dE/dD at fixed R~ equals D^-T V  (all 9 components; exact, no factor issue)
    rng = np.random.default_rng(20 + kind)
    Rt, h0, D, pot, rc = system(kind, rng)
    E, F, V = E_of(Rt, h0, D, kind, pot, rc)
    Gc = cf.generalized_force(F, V, D, 1.0, cf.CELL_D)[-3:]
    eps = 1e-6
    for m in range(3):
        for n in range(3):
            dD = np.zeros((3, 3))
            dD[m, n] = eps
            fd = -(E_of(Rt, h0, D + dD, kind, pot, rc)[0] - E_of(Rt, h0, D - dD, kind, pot, rc)[0]) / (2 * eps)
            assert abs(fd - Gc[m, n]) < 1e-6 * np.abs(Gc).max()


@pytest.mark.parametrize("kind", [0, 1])
def test_rotation_free_force_eq16_eq17_factor_two(kind):
    # Reading A9: Eq. 17 as printed, (D^-T V D^-1) : S = -2 dE/d eta for E(B + eta S), S symmetric, D = sqrt(B).
    rng = np.random.default_rng(30 + kind)
    Rt, h0, D, pot, rc = system(kind, rng)
    B = D @ D.T
    Ds = cf.cell_map(B)
    E, F, V = E_of(Rt, h0, Ds, kind, pot, rc)
    Gc = cf.generalized_force(F, V, Ds, 1.0, cf.CELL_B)[-3:]
    assert np.allclose(Gc, Gc.T, atol=1e-10 * np.abs(Gc).max())
    eta = 1e-6
    for trial in range(3):
        S = rng.standard_normal((3, 3))
        S = 0.5 * (S + S.T)
        Ep = E_of(Rt, h0, cf.cell_map(B + eta * S), kind, pot, rc)[0]
        Em = E_of(Rt, h0, cf.cell_map(B - eta * S), kind, pot, rc)[0]
        fd = -(Ep - Em) / (2 * eta)
        assert abs(np.sum(Gc * S) - 2.0 * fd) < 2e-6 * np.abs(Gc).max()
    # lam scales the cell block by 1/lam
    assert np.allclose(cf.generalized_force(F, V, Ds, 4.0, cf.CELL_B)[-3:], Gc / 4.0)


@pytest.mark.parametrize("kind", [0, 1])
def test_rotation_invariance_p110_p124(kind):
    # under (R, h) -> (R Q, h Q): R~, B, F D^T and D^-T V D^-1 are unchanged; D^-T V (Eq. 14) is not.
    rng = np.random.default_rng(40 + kind)
    Rt, h0, D, pot, rc = system(kind, rng)
    Q, _ = np.linalg.qr(rng.standard_normal((3, 3)))
    if np.linalg.det(Q) < 0:
        Q[:, 0] *= -1
    out = []
    for rot in (np.eye(3), Q):
        R, h = (Rt @ D) @ rot, (h0 @ D) @ rot
        Rt_, B_, D_ = cf.input_mapping(R, h, h0)
        nb = ff.neighbors(Rt_, h0, h, rc, 400, brute=True)
        E, F, V = ff.energy_force_virial(Rt_, h0, h, kind, pot, nb)
        GB = cf.generalized_force(F, V, D_, 1.0, cf.CELL_B)
        GD = cf.generalized_force(F, V, D_, 1.0, cf.CELL_D)
        out.append((Rt_, B_, GB, GD, E))
    a, b = out
    assert np.allclose(a[0], b[0], atol=1e-12) and np.allclose(a[1], b[1], atol=1e-12)
    assert np.abs(a[2] - b[2]).max() < 1e-11 * np.abs(a[2]).max()
    assert abs(a[4] - b[4]) < 1e-11 * abs(a[4])
    assert np.abs(a[3][-3:] - b[3][-3:]).max() > 1e-3 * np.abs(a[3][-3:]).max()
    # and the rotation-free path: evaluating at D = sqrt(B) gives the same energy as the rotated input
    Ds = cf.cell_map(a[1])
    assert abs(E_of(a[0], h0, Ds, kind, pot, rc)[0] - a[4]) < 1e-11 * abs(a[4])


def test_cell_map_is_the_symmetric_positive_root():
    rng = np.random.default_rng(7)
    for _ in range(5):
        D = np.eye(3) + 0.3 * rng.standard_normal((3, 3))
        B = D @ D.T
        S = cf.cell_map(B)
        assert np.allclose(S @ S, B, atol=1e-13) and np.allclose(S, S.T, atol=1e-15)
        assert np.all(np.linalg.eigvalsh(S) > 0)
        Dsym = 0.5 * (D + D.T) + 2 * np.eye(3)  # symmetric PD: sqrt(D^2) = D
        assert np.allclose(cf.cell_map(Dsym @ Dsym), Dsym, atol=1e-13)
    with pytest.raises(ValueError):
        cf.cell_map(np.diag([1.0, -0.1, 1.0]))


def test_pack_unpack():
    Rt = np.arange(12.0).reshape(4, 3)
    B = np.diag([1.0, 2.0, 3.0])
    X = cf.pack(Rt, B, 2.5)
    assert X.shape == (7, 3) and np.allclose(X[-3:], 2.5 * B)
    Rt2, B2 = cf.unpack(X, 2.5)
    assert np.array_equal(Rt2, Rt) and np.allclose(B2, B)
