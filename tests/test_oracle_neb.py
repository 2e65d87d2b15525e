"""Pins for oracle/neb.py: improved tangent (ref [13]), Eq. 1 + climbing image (ref [12]), FIRE (O7),
and CI-NEB on the analytic Mueller-Brown surface reproducing its saddle energies to 1e-6
(BASELINE.json north_star)."""
import os

import numpy as np
import pytest

from oracle import mullerbrown as mb
from oracle.neb import Band, Fire, improved_tangent, neb_force

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "mueller_brown_stationary_points.txt")


def golden_points():
    pts = []
    with open(GOLDEN) as fh:
        for line in fh:
            if line.startswith("#") or not line.strip():
                continue
            kind, x, y, v = line.split()
            pts.append((kind, float(x), float(y), float(v)))
    return pts


# ---------- Mueller-Brown surface itself: independent Newton iteration on grad V = 0 ----------

def mb_value_grad_hess(x, y):
    """Independent restatement (test-side) with analytic Hessian, used only to locate stationary points."""
    A = [-200.0, -100.0, -170.0, 15.0]
    a = [-1.0, -1.0, -6.5, 0.7]
    b = [0.0, 0.0, 11.0, 0.6]
    c = [-10.0, -10.0, -6.5, 0.7]
    X0 = [1.0, 0.0, -0.5, -1.0]
    Y0 = [0.0, 0.5, 1.5, 1.0]
    V, g, H = 0.0, np.zeros(2), np.zeros((2, 2))
    for k in range(4):
        dx, dy = x - X0[k], y - Y0[k]
        e = A[k] * np.exp(a[k] * dx * dx + b[k] * dx * dy + c[k] * dy * dy)
        ux, uy = 2 * a[k] * dx + b[k] * dy, b[k] * dx + 2 * c[k] * dy
        V += e
        g += e * np.array([ux, uy])
        H += e * (np.outer([ux, uy], [ux, uy]) + np.array([[2 * a[k], b[k]], [b[k], 2 * c[k]]]))
    return V, g, H


def test_mueller_brown_golden_points_are_stationary_and_oracle_surface_agrees():
    for kind, x, y, v in golden_points():
        p = np.array([x, y])
        for _ in range(20):
            V, g, H = mb_value_grad_hess(*p)
            p = p - np.linalg.solve(H, g)
        V, g, H = mb_value_grad_hess(*p)
        assert np.abs(p - [x, y]).max() < 2e-6 and abs(V - v) < 1e-7
        w = np.linalg.eigvalsh(H)
        assert (w[0] < 0 < w[1]) if kind == "saddle" else (w[0] > 0)
        Vo, Fo = mb.energy_force(p)
        assert abs(Vo - V) < 1e-12 and np.abs(Fo).max() < 1e-8
    # oracle force = -grad V by finite differences at a generic point
    q, eps = np.array([-0.3, 0.9]), 1e-6
    V0, F0 = mb.energy_force(q)
    for m in range(2):
        d = np.zeros(2)
        d[m] = eps
        fd = -(mb.energy_force(q + d)[0] - mb.energy_force(q - d)[0]) / (2 * eps)
        assert abs(fd - F0[m]) < 1e-6 * np.abs(F0).max()


MB_FIRE = dict(dt0=2e-4, dtmax=4e-3, maxstep=0.05, nmin=5, finc=1.1, fdec=0.5, astart=0.1, fa=0.99)


@pytest.mark.parametrize("a,b,saddle", [(0, 2, 3), (2, 1, 4)])
def test_ci_neb_reproduces_mueller_brown_saddle_energies(a, b, saddle):
    pts = golden_points()
    A, B, S = np.array(pts[a][1:3]), np.array(pts[b][1:3]), pts[saddle]
    P = 11
    X = [(A + (B - A) * p / (P - 1)).reshape(1, 2) for p in range(P)]
    band = Band(X, mb.eval_images, k_spring=50.0, climb=True, fire=MB_FIRE)
    band.run(1e-5, 20000)
    assert band.fmax < 1e-5
    assert abs(band.E[band.pstar] - S[3]) < 1e-6
    assert np.abs(band.X[band.pstar].ravel() - S[1:3]).max() < 1e-5
    assert abs(band.barrier - (S[3] - pts[a][3])) < 1e-4  # endpoints given to 6 digits
    # without the climbing image the highest image only brackets the saddle from below
    band2 = Band(X, mb.eval_images, k_spring=50.0, climb=False, fire=MB_FIRE)
    band2.run(1e-4, 20000)
    assert band2.E.max() <= S[3] + 1e-6


# ---------- tangent ----------

def test_improved_tangent_branches_and_continuity():
    rng = np.random.default_rng(0)
    Xm, X, Xp = rng.standard_normal((3, 4, 3))
    tp, tm = Xp - X, X - Xm
    assert np.array_equal(improved_tangent(Xm, X, Xp, 0.0, 1.0, 2.0)[0], tp)  # uphill: forward difference
    assert np.array_equal(improved_tangent(Xm, X, Xp, 2.0, 1.0, 0.0)[0], tm)  # downhill: backward difference
    # maximum, E_next > E_prev: tau+ dEmax + tau- dEmin
    tau = improved_tangent(Xm, X, Xp, 0.0, 1.0, 0.4)[0]
    assert np.allclose(tau, tp * 1.0 + tm * 0.6)
    tau = improved_tangent(Xm, X, Xp, 0.4, 1.0, 0.0)[0]
    assert np.allclose(tau, tp * 0.6 + tm * 1.0)
    # minimum
    tau = improved_tangent(Xm, X, Xp, 3.0, 1.0, 1.5)[0]
    assert np.allclose(tau, tp * 0.5 + tm * 2.0)
    # continuity across the branch switches (O5): E -> E_next from either side
    e = 1e-12
    t1 = improved_tangent(Xm, X, Xp, 0.0, 1.0 - e, 1.0)[0]  # monotone: tau+
    t2 = improved_tangent(Xm, X, Xp, 0.0, 1.0 + e, 1.0)[0]  # maximum with dEmin -> 0
    assert np.abs(t1 / np.linalg.norm(t1) - t2 / np.linalg.norm(t2)).max() < 1e-10
    # A26: three exactly equal energies (the weights of ref [13] both vanish): the bisector, never a zero tangent;
    # one equal neighbour is still the ordinary extremum branch with dEmin = 0
    assert np.array_equal(improved_tangent(Xm, X, Xp, 1.0, 1.0, 1.0)[0], tp + tm)
    assert np.allclose(improved_tangent(Xm, X, Xp, 1.0, 1.0, 0.5)[0], tm * 0.5)
    assert np.allclose(improved_tangent(Xm, X, Xp, 0.5, 1.0, 1.0)[0], tp * 0.5)
    f = neb_force(rng.standard_normal((4, 3)), *improved_tangent(Xm, X, Xp, 1.0, 1.0, 1.0), 1.0, climbing=False)
    assert np.all(np.isfinite(f))


# ---------- Eq. 1 ----------

def test_neb_force_projection_identities():
    rng = np.random.default_rng(1)
    G, tau, tp, tm = rng.standard_normal((4, 5, 3))
    t = tau / np.linalg.norm(tau)
    k = 1.7
    f = neb_force(G, tau, tp, tm, k, climbing=False)
    spring = k * (np.linalg.norm(tp) - np.linalg.norm(tm))
    assert abs(np.sum((f - spring * t) * t)) < 1e-13  # (f - f_spring) . t = 0
    assert abs(np.sum(f * t) - spring) < 1e-13  # f . t = spring magnitude
    assert np.allclose(f - spring * t, G - np.sum(G * t) * t)  # perpendicular part of the true force
    fc = neb_force(G, tau, tp, tm, k, climbing=True)
    assert abs(np.sum(fc * t) + np.sum(G * t)) < 1e-13  # climbing: parallel component inverted
    assert np.allclose(fc - np.sum(fc * t) * t, G - np.sum(G * t) * t)  # perpendicular part untouched
    with pytest.raises(ValueError):
        neb_force(G, np.zeros_like(G), tp, tm, k, False)


# ---------- FIRE ----------

def test_fire_on_1d_harmonic_hand_computed():
    # U = x^2/2, f = -x.  Step 1 (A2: no power test): v = dt f, x1 = x0 (1 - dt^2).
    dt = 0.1
    fire = Fire((1, 1, 1), dt0=dt, dtmax=1.0, maxstep=10.0, nmin=5, finc=1.1, fdec=0.5, astart=0.1, fa=0.99)
    x = 1.0
    x += fire.step(np.full((1, 1, 1), -x), 1).item()
    assert abs(x - (1 - dt * dt)) < 1e-15 and fire.dt == dt
    # Step 2: power = f.v > 0; 1-D mixing leaves v unchanged ((1-a)v + a|v| f/|f| = v); v += dt f
    v1 = -dt * 1.0
    f2 = -x
    v2 = v1 + dt * f2
    x2 = x + dt * v2
    x += fire.step(np.full((1, 1, 1), f2), 1).item()
    assert abs(x - x2) < 1e-15 and fire.n_pos == 1 and fire.dt == dt
    # overshoot: force opposes velocity -> v zeroed, dt halved, alpha reset
    fire.v[:] = 1.0
    d = fire.step(np.full((1, 1, 1), -2.0), 1).item()
    assert fire.dt == dt * 0.5 and fire.n_pos == 0 and fire.alpha == 0.1
    assert abs(d - (fire.dt * (fire.dt * -2.0))) < 1e-15


def test_fire_dt_growth_and_step_clip():
    fire = Fire((1, 2, 1), dt0=0.1, dtmax=0.15, maxstep=0.01, nmin=2, finc=1.1, fdec=0.5, astart=0.1, fa=0.99)
    f = np.array([1.0, 1.0]).reshape(1, 2, 1)
    dts = []
    for _ in range(10):
        d = fire.step(f, 2)
        dts.append(fire.dt)
        assert np.linalg.norm(d) <= 0.01 * np.sqrt(2) * (1 + 1e-12)  # |Delta|_2 <= maxstep sqrt(rows)
    # n_pos reaches nmin+1 after the 4th step (first step skipped): dt grows by 1.1 per step, capped at dtmax
    assert dts[:4] == [0.1, 0.1, 0.1, 0.1] and abs(dts[4] - 0.11) < 1e-15
    assert abs(dts[7] - 0.1 * 1.1 ** 4) < 1e-15 and dts[-1] == 0.15


def test_fire_converges_on_anisotropic_quadratic_and_clip_inactive_is_identity():
    K = np.array([1.0, 25.0, 4.0])
    def run(maxstep):
        fire = Fire((1, 1, 3), dt0=0.05, dtmax=0.3, maxstep=maxstep)
        x = np.array([1.0, -0.5, 0.7]).reshape(1, 1, 3)
        for it in range(2000):
            f = -K * x
            if np.abs(f).max() < 1e-10:
                break
            x = x + fire.step(f, 1)
        return x, it
    x, it = run(1e9)
    assert np.abs(x).max() < 1e-10 and it < 1000
    x2, it2 = run(5.0)  # clip never active => identical trajectory
    assert it2 == it and np.array_equal(x, x2)
