"""Pins for the external-pressure reading A25 (oracle/cfneb.py): H = U + p Omega, V_H = V - p Omega I.

The paper's graphite band is "under 40GPa" (Fig. 3 caption) with no equations; Eq. 2-3 (right-multiplied
strain, V = -dU/d eps) fix what a hydrostatic pressure adds.  Pinned by (i) finite differences of an enthalpy the
test assembles itself (U from the p = 0 oracle, already pinned, + p |det h| computed here), (ii) the textbook
equilibrium condition: a cell relaxed under p has internal pressure tr V / (3 Omega) = p, (iii) p = 0 changes nothing.
"""
import numpy as np

from cfneb_workloads import fcc_supercell, lj_params
from oracle import cellfilter as cf
from oracle import cfneb as oc
from oracle import forcefield as ff

P_EXT = 0.7  # eps / sigma^3


def _system():
    rng = np.random.default_rng(5)
    frac, h0 = fcc_supercell(2, 2, 2, 1.56)
    h0 = h0 @ (np.eye(3) + 0.02 * rng.standard_normal((3, 3)))
    Rt = frac @ h0 + 0.03 * rng.standard_normal(frac.shape)
    return Rt, h0


def test_cell_force_is_minus_dH_dD_by_finite_differences():
    Rt, h0 = _system()
    lam = 1.3
    D = np.eye(3) + 0.04 * np.random.default_rng(6).standard_normal((3, 3))
    ev_p = oc.CrystalEvaluator(h0, 0, lj_params(), 2.8, 400, lam, cf.CELL_D, brute=True, pressure=P_EXT)
    ev_0 = oc.CrystalEvaluator(h0, 0, lj_params(), 2.8, 400, lam, cf.CELL_D, brute=True, pressure=0.0)

    def H(Dm):  # enthalpy assembled by the test: U of the p = 0 evaluator + p |det(h0 D)|
        U = ev_0([cf.pack(Rt, Dm, lam)])[0][0]
        return U + P_EXT * abs(np.linalg.det(h0 @ Dm))

    E, G = ev_p([cf.pack(Rt, D, lam)])
    assert abs(E[0] - H(D)) < 1e-12 * abs(E[0])
    eps = 1e-6
    for a in range(3):
        for b in range(3):
            Dp, Dm = D.copy(), D.copy()
            Dp[a, b] += eps
            Dm[a, b] -= eps
            fd = -(H(Dp) - H(Dm)) / (2 * eps) / lam  # coordinate is lam * D
            assert abs(fd - G[0][-3 + a, b]) < 2e-7 * np.abs(G[0][-3:]).max(), (a, b)
    # the pressure term is not small here: dropping it must fail the check above
    G0 = ev_0([cf.pack(Rt, D, lam)])[1][0]
    assert np.abs(G0[-3:] - G[0][-3:]).max() > 1e-2 * np.abs(G[0][-3:]).max()
    # atom rows do not see the pressure
    assert np.array_equal(G0[:-3], G[0][:-3])


def test_relaxed_cell_carries_the_external_pressure():
    frac, h0 = fcc_supercell(2, 2, 2, 1.56)
    R = frac @ h0
    out = {}
    for p in (0.0, P_EXT):
        Rr, hr, E, fmax, it = oc.relax_endpoint(R, h0, 0, lj_params(), 2.5, fmax_tol=1e-9, max_steps=4000, pressure=p)
        assert fmax < 1e-9
        nb = ff.neighbors(Rr @ np.linalg.inv(np.linalg.solve(h0, hr)), h0, hr, 2.5, 400)
        U, F, V = ff.energy_force_virial(Rr @ np.linalg.inv(np.linalg.solve(h0, hr)), h0, hr, 0, lj_params(), nb)
        omega = abs(np.linalg.det(hr))
        out[p] = (omega, np.trace(V) / (3.0 * omega), U, E)
    assert abs(out[0.0][1]) < 1e-8                      # stress-free at p = 0
    assert abs(out[P_EXT][1] - P_EXT) < 1e-8            # internal pressure tr V / (3 Omega) = p
    assert out[P_EXT][0] < out[0.0][0]                  # compressed
    assert abs(out[P_EXT][3] - (out[P_EXT][2] + P_EXT * out[P_EXT][0])) < 1e-10 * abs(out[P_EXT][3])  # E returned is H


def test_zero_pressure_is_the_plain_band():
    from cfneb_workloads import build_workload
    spec, pos, cells = build_workload(0)
    kw = dict(k_spring=spec.k_spring, climb=True, cell_factor=0.0, fire=spec.fire, skin=spec.skin,
              max_neighbors=spec.max_neighbors)
    a = oc.CFNEB(pos, cells, spec.potential, spec.pot, spec.r_cut, **kw)
    b = oc.CFNEB(pos, cells, spec.potential, spec.pot, spec.r_cut, pressure=0.0, **kw)
    a.step(3)
    b.step(3)
    assert np.array_equal(a.get_state()[0], b.get_state()[0])
    c = oc.CFNEB(pos, cells, spec.potential, spec.pot, spec.r_cut, pressure=P_EXT, **kw)
    c.step(3)
    assert not np.allclose(c.get_state()[0][:, -3:], a.get_state()[0][:, -3:], atol=1e-6)  # cells respond to p
