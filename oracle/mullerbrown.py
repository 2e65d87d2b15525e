"""Analytic 2-D Mueller-Brown surface -- CPU ORACLE, TEST INFRASTRUCTURE ONLY.

Pin for oracle/neb.py (BASELINE.json north_star: "CI-NEB on the analytic 2-D Mueller-Brown surface
reproducing its known saddle energies to 1e-6").  Standard parameters (K. Mueller, L. D. Brown,
Theor. Chim. Acta 53, 75 (1979)):  V = sum_k A_k exp[a_k (x-x0_k)^2 + b_k (x-x0_k)(y-y0_k) + c_k (y-y0_k)^2].
"""
import numpy as np

A = np.array([-200.0, -100.0, -170.0, 15.0])
a = np.array([-1.0, -1.0, -6.5, 0.7])
b = np.array([0.0, 0.0, 11.0, 0.6])
c = np.array([-10.0, -10.0, -6.5, 0.7])
x0 = np.array([1.0, 0.0, -0.5, -1.0])
y0 = np.array([0.0, 0.5, 1.5, 1.0])


def energy_force(xy):
    """V and force -grad V at the point xy (shape (2,) or (1,2))."""
    x, y = float(np.ravel(xy)[0]), float(np.ravel(xy)[1])
    dx, dy = x - x0, y - y0
    e = A * np.exp(a * dx * dx + b * dx * dy + c * dy * dy)
    V = float(np.sum(e))
    gx = float(np.sum(e * (2.0 * a * dx + b * dy)))
    gy = float(np.sum(e * (b * dx + 2.0 * c * dy)))
    return V, -np.array([gx, gy])


def eval_images(X_list):
    """Band callback: each X is a (1, 2) array (one row of two dofs)."""
    E, G = [], []
    for X in X_list:
        V, F = energy_force(X)
        E.append(V)
        G.append(F.reshape(np.shape(X)))
    return E, G
