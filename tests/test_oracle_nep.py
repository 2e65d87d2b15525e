"""Pins of the NEP-shaped potential of the oracle (kind 4; "NEP-trained force field", the shape of the
paper's force field with seeded weights): site energies rebuilt from numpy's Chebyshev / Legendre routines, a dense
product and tanh with an independent SplitMix64 weight stream; finite differences of forces and of all nine virial
components; rotation / translation invariance; the two cut-offs and the two atom types each change the result."""
import numpy as np
import pytest
from numpy.polynomial import chebyshev as Ch
from numpy.polynomial import legendre as Le

from cfneb_workloads import nep_params
from oracle import forcefield as ff

M64 = (1 << 64) - 1


def splitmix(seed):
    st = int(seed)
    while True:
        st = (st + 0x9E3779B97F4A7C15) & M64
        z = st
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & M64
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & M64
        z ^= z >> 31
        yield 2.0 * ((z >> 11) / 9007199254740992.0) - 1.0


def weights(pot):
    """The weight stream in the order include/cfneb.h states."""
    rcr, rca, nr, na, kr, ka, L, H, T, seed = [pot[0], pot[1]] + [int(x) for x in pot[2:10]]
    D = nr + na * L
    g = splitmix(seed)
    W0, b0, W1 = np.zeros((T, H, D)), np.zeros((T, H)), np.zeros((T, H))
    for I in range(T):
        for mu in range(H):
            for d in range(D):
                W0[I, mu, d] = next(g) * (0.04 if d < nr else 0.004)
        for mu in range(H):
            b0[I, mu] = 0.5 * next(g)
        for mu in range(H):
            W1[I, mu] = next(g)
    cR = np.array([next(g) for _ in range(T * T * nr * kr)]).reshape(T, T, nr, kr)
    cA = np.array([next(g) for _ in range(T * T * na * ka)]).reshape(T, T, na, ka)
    return W0, b0, W1, cR, cA


def basis(r, rc, K):
    """f_k(r) = 1/2 [T_k(x) + 1] fc(r), from numpy's Chebyshev evaluation."""
    x = 2.0 * (r / rc - 1.0) ** 2 - 1.0
    fc = 0.5 * (1.0 + np.cos(np.pi * r / rc))
    return np.array([0.5 * (Ch.chebval(x, [0] * k + [1]) + 1.0) * fc for k in range(K)])


def site_energies(R, types, pot):
    """The definition, written with library routines: no periodic images (an isolated cluster)."""
    rcr, rca, nr, na, kr, ka, L, H, T, seed = [pot[0], pot[1]] + [int(x) for x in pot[2:10]]
    W0, b0, W1, cR, cA = weights(pot)
    N = len(R)
    U = np.zeros(N)
    for i in range(N):
        I = types[i]
        q = np.zeros(nr + na * L)
        env = []
        for j in range(N):
            if j == i:
                continue
            d = R[j] - R[i]
            r = np.linalg.norm(d)
            if r < rcr:
                q[:nr] += cR[I, types[j]] @ basis(r, rcr, kr)
            if r < rca:
                env.append((d / r, cA[I, types[j]] @ basis(r, rca, ka)))
        for (ua, ga) in env:
            for (ub, gb) in env:
                c = float(np.dot(ua, ub))
                for l in range(1, L + 1):
                    q[nr + np.arange(na) * L + l - 1] += ga * gb * Le.legval(c, [0] * l + [1])
        U[i] = W1[I] @ np.tanh(W0[I] @ q - b0[I])
    return U


def cluster(seed=3, n=9):
    rng = np.random.default_rng(seed)
    R = rng.uniform(-2.2, 2.2, size=(n, 3))
    R += 20.0  # inside a big box: no periodic images within the cut-off
    types = (np.arange(n) % 2).astype(np.int32)
    types[3] = 0
    return R, types, np.eye(3) * 40.0


def evaluate(R, cell, types, pot, cap=64, per_atom=False):
    ff.set_types(types)
    nb = ff.neighbors(R, cell, cell, pot[0], cap)
    out = ff.energy_force_virial(R, cell, cell, 4, pot, nb, per_atom=per_atom)
    ff.set_types(None)
    return out


POT = nep_params(rc_r=3.9, rc_a=2.9, n_r=3, n_a=2, k_r=5, k_a=4, L=4, H=7, n_types=2, seed=1234567)


def test_site_energies_equal_the_definition_written_with_library_polynomials():
    R, types, cell = cluster()
    E, F, V, Ui, _ = evaluate(R, cell, types, POT, per_atom=True)
    U_ref = site_energies(R, types, POT)
    assert np.abs(Ui - U_ref).max() < 1e-12 and abs(E - U_ref.sum()) < 1e-12
    assert np.abs(U_ref).max() > 1e-2                       # not a trivially small number
    # both cut-offs matter: some neighbours lie between rc_a and rc_r, some inside rc_a
    d = np.linalg.norm(R[:, None] - R[None], axis=2)
    assert np.any((d > POT[1]) & (d < POT[0])) and np.any((d > 0) & (d < POT[1]))
    # ... and so do the types: one species only gives other energies
    E1 = evaluate(R, cell, np.zeros(len(R), dtype=np.int32), POT)[0]
    assert abs(E1 - E) > 1e-3
    assert abs(E1 - site_energies(R, np.zeros(len(R), dtype=int), POT).sum()) < 1e-12
    # other shapes exercise the index arithmetic (L < 4, one type, k_r != k_a, H large)
    for kw in (dict(L=1, H=3), dict(n_types=1, n_r=8, n_a=1, k_r=12, k_a=2), dict(L=3, H=40, n_r=1, n_a=5)):
        base = dict(rc_r=3.9, rc_a=2.9, n_r=3, n_a=2, k_r=5, k_a=4, L=4, H=7, n_types=2, seed=99)
        base.update(kw)
        pot = nep_params(**base)
        t = types if base["n_types"] == 2 else np.zeros(len(R), dtype=np.int32)
        assert abs(evaluate(R, cell, t, pot)[0] - site_energies(R, t, pot).sum()) < 1e-12


def test_forces_and_virial_by_finite_differences():
    """Eq. 5 (F = -dE/dR) and Eq. 3 / 8 (V = -dE/d eps under h -> h (I + eps), fractional coordinates fixed) on a
    periodic two-species cell whose box is narrower than 2 rc_r (atoms see several images of one neighbour)."""
    rng = np.random.default_rng(11)
    cell = np.array([[5.1, 0.2, -0.1], [0.3, 4.7, 0.15], [-0.2, 0.1, 5.4]])
    frac = rng.uniform(0, 1, size=(14, 3))
    types = (np.arange(14) % 2).astype(np.int32)
    pot = nep_params(rc_r=3.4, rc_a=2.8, n_r=3, n_a=2, k_r=4, k_a=4, L=4, H=6, n_types=2, seed=42)
    R = frac @ cell
    E, F, V = evaluate(R, cell, types, pot, cap=200)
    hh = 1e-5
    for (i, m) in ((0, 0), (5, 1), (13, 2), (7, 0)):
        Rp, Rm = R.copy(), R.copy()
        Rp[i, m] += hh
        Rm[i, m] -= hh
        fd = -(evaluate(Rp, cell, types, pot, cap=200)[0] - evaluate(Rm, cell, types, pot, cap=200)[0]) / (2 * hh)
        assert abs(fd - F[i, m]) < 2e-7 * max(1.0, np.abs(F).max()), (i, m, fd, F[i, m])
    assert np.abs(F.sum(axis=0)).max() < 1e-11
    for a in range(3):
        for b in range(3):
            eps = np.zeros((3, 3))
            eps[a, b] = hh
            Ep = evaluate(frac @ (cell @ (np.eye(3) + eps)), cell @ (np.eye(3) + eps), types, pot, cap=200)[0]
            Em = evaluate(frac @ (cell @ (np.eye(3) - eps)), cell @ (np.eye(3) - eps), types, pot, cap=200)[0]
            assert abs(-(Ep - Em) / (2 * hh) - V[a, b]) < 2e-7 * max(1.0, np.abs(V).max()), (a, b)
    assert np.abs(V - V.T).max() < 1e-10 * np.abs(V).max()


def test_rotation_and_translation_invariance():
    R, types, cell = cluster(seed=8, n=11)
    E, F, V = evaluate(R, cell, types, POT)
    Q, _ = np.linalg.qr(np.random.default_rng(2).standard_normal((3, 3)))
    if np.linalg.det(Q) < 0:
        Q[:, 0] *= -1
    c = R.mean(axis=0)
    R2 = (R - c) @ Q + c + np.array([0.3, -0.2, 0.1])
    E2, F2, V2 = evaluate(R2, cell, types, POT)
    assert abs(E2 - E) < 1e-11
    assert np.abs(F2 - F @ Q).max() < 1e-10 and np.abs(V2 - Q.T @ V @ Q).max() < 1e-10


def test_parameter_errors():
    R, types, cell = cluster()
    for bad in (dict(L=5), dict(n_r=9), dict(k_a=13), dict(H=65), dict(n_types=3), dict(rc_a=4.5)):
        base = dict(rc_r=3.9, rc_a=2.9, n_r=3, n_a=2, k_r=5, k_a=4, L=4, H=7, n_types=2, seed=1)
        base.update(bad)
        with pytest.raises(ff.OracleError):
            evaluate(R, cell, types, nep_params(**base))
