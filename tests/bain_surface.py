"""Closed-form energy per atom of a perfect body-centred tetragonal crystal E(a, c) for the Finnis-Sinclair-type
potential of BASELINE.json configs[2-4], by a direct lattice sum (numpy, no neighbour lists, no oracle code), and
its saddle between bcc (c/a = 1) and the c/a = sqrt(2) end state by Newton's method on the 2-D surface.

Used to pin the Bain bands: a homogeneous transformation of a perfect crystal has the same barrier per atom in any
supercell, and that barrier is the saddle of this two-variable function -- a number that involves no tangent, no
projection, no cell filter and no optimizer.
"""
import numpy as np


def energy_per_atom(a, c, pot):
    D, alpha, r0, beta, rr0, A, r_on, r_cut = [float(x) for x in pot[:8]]
    rng = np.arange(-5, 6)
    g = np.stack(np.meshgrid(rng, rng, rng, indexing="ij"), -1).reshape(-1, 3).astype(np.float64)
    pts = np.concatenate([g, g + 0.5]) * np.array([a, a, c])
    r = np.linalg.norm(pts, axis=1)
    r = r[(r > 1e-9) & (r < r_cut)]
    t = np.where(r <= r_on, 1.0, 0.5 * (1.0 + np.cos(np.pi * (r - r_on) / (r_cut - r_on))))
    v = D * (np.exp(-2.0 * alpha * (r - r0)) - 2.0 * np.exp(-alpha * (r - r0))) * t
    rho = np.sum(np.exp(-beta * (r - rr0)) * t)
    return 0.5 * np.sum(v) - A * np.sqrt(rho)


def saddle(a, c, pot, d=1e-4, iters=12):
    """Newton on grad E(a, c) = 0 from the guess (a, c).  Returns (a*, c*, E*, Hessian eigenvalues)."""
    x = np.array([a, c], dtype=np.float64)
    f = lambda y: energy_per_atom(y[0], y[1], pot)

    def grad_hess(x):
        g, H = np.zeros(2), np.zeros((2, 2))
        for i in range(2):
            e = np.zeros(2)
            e[i] = d
            g[i] = (f(x + e) - f(x - e)) / (2 * d)
            for j in range(2):
                e2 = np.zeros(2)
                e2[j] = d
                H[i, j] = (f(x + e + e2) - f(x + e - e2) - f(x - e + e2) + f(x - e - e2)) / (4 * d * d)
        return g, H

    for _ in range(iters):
        g, H = grad_hess(x)
        x = x - np.linalg.solve(H, g)
    g, H = grad_hess(x)
    assert np.abs(g).max() < 1e-9
    return x[0], x[1], f(x), np.linalg.eigvalsh(H)
