"""Generic NEB + FIRE over a band of n-dof points -- CPU ORACLE, TEST INFRASTRUCTURE ONLY.

The paper states Eq. 1, f^NEB = f^real|_perp + f^spring, and cites the improved tangent
(ref [13]) and the climbing image (ref [12]) without printing formulas.
The optimizer is unnamed in the paper ("standard optimizers"); FIRE is fixed by
BASELINE.json north_star.  Formulas below are SURVEY.md §8(c) O5-O8 with readings A1-A6.

Generic over the energy/force callback so the same code runs on the 2-D Mueller-Brown surface
(n = 2, the pin) and on crystals (n = 3N + 9, generalized coordinates of the cell filter).
"""
import numpy as np


def improved_tangent(X_prev, X, X_next, E_prev, E, E_next):
    """O5 (ref [13]): upwind tangent.  Returns (tau, tau_plus, tau_minus), tau NOT normalised."""
    tp = X_next - X
    tm = X - X_prev
    if E_next > E > E_prev:
        tau = tp
    elif E_next < E < E_prev:
        tau = tm
    else:
        dmax = max(abs(E_next - E), abs(E_prev - E))
        dmin = min(abs(E_next - E), abs(E_prev - E))
        if dmax == 0.0:
            # A26: E_prev == E == E_next exactly (three images at the bottom of one basin, which a long band of a
            # perfect crystal produces): both weights vanish and ref [13] defines no tangent; take the bisector.
            tau = tp + tm
        elif E_next > E_prev:
            tau = tp * dmax + tm * dmin
        else:  # includes the tie E_next == E_prev
            tau = tp * dmin + tm * dmax
    return tau, tp, tm


def neb_force(G, tau, tp, tm, k_spring, climbing):
    """O6 (Eq. 1; reading A6): f = G - (G.t)t + k(|tau+| - |tau-|) t;  climbing: f = G - 2 (G.t) t."""
    nt = np.sqrt(np.sum(tau * tau))
    if nt == 0.0:
        raise ValueError("zero tangent")
    t = tau / nt
    Gt = np.sum(G * t)
    if climbing:
        return G - 2.0 * Gt * t
    spring = k_spring * (np.sqrt(np.sum(tp * tp)) - np.sqrt(np.sum(tm * tm)))
    return G - Gt * t + spring * t


class Fire:
    """O7: FIRE with one state for the whole band (readings A1-A4)."""

    def __init__(self, shape, dt0=0.1, dtmax=1.0, maxstep=0.2, nmin=5, finc=1.1, fdec=0.5, astart=0.1, fa=0.99):
        self.dt0, self.dtmax, self.maxstep = dt0, dtmax, maxstep
        self.nmin, self.finc, self.fdec, self.astart, self.fa = nmin, finc, fdec, astart, fa
        self.shape = shape
        self.reset()

    def reset(self):
        self.v = np.zeros(self.shape)
        self.dt = self.dt0
        self.alpha = self.astart
        self.n_pos = 0
        self.first = True

    def step(self, f, n_rows):
        """One FIRE step for force f (same shape as v); returns the displacement Delta.

        n_rows = number of movable rows (M (N+3) for crystals): the global 2-norm of Delta is
        limited to maxstep * sqrt(n_rows) (A4).
        """
        if self.first:
            self.first = False  # A2: skip the power test on the first step (v = 0)
        else:
            power = np.sum(f * self.v)
            if power > 0.0:
                nv = np.sqrt(np.sum(self.v * self.v))
                nf = np.sqrt(np.sum(f * f))
                self.v = (1.0 - self.alpha) * self.v + self.alpha * (nv / nf) * f
                if self.n_pos > self.nmin:
                    self.dt = min(self.dt * self.finc, self.dtmax)
                    self.alpha = self.alpha * self.fa
                self.n_pos += 1
            else:
                self.v = np.zeros(self.shape)
                self.alpha = self.astart
                self.dt = self.dt * self.fdec
                self.n_pos = 0
        self.v = self.v + self.dt * f  # unit mass
        delta = self.dt * self.v
        limit = self.maxstep * np.sqrt(n_rows)
        nd = np.sqrt(np.sum(delta * delta))
        if nd > limit:
            delta = delta * (limit / nd)
        return delta


class Band:
    """A chain of P points X[p] (each an (rows, row_len) array), endpoints fixed.

    eval_images(X_list) -> (E list, G list): energies and generalized forces of the given points.
    post_update(X) -> X: hook applied to each updated point (crystals: symmetrise B, O7 step 4).
    """

    def __init__(self, X, eval_images, k_spring=1.0, climb=True, fire=None, post_update=None):
        self.X = [np.array(x, dtype=np.float64) for x in X]
        self.P = len(self.X)
        self.eval_images = eval_images
        self.k = k_spring
        self.climb = climb
        self.post_update = post_update
        M = self.P - 2
        self.fire = Fire((M,) + self.X[0].shape, **(fire or {}))
        E, _ = eval_images([self.X[0], self.X[-1]])
        self.E = np.zeros(self.P)
        self.E[0], self.E[-1] = E[0], E[1]
        self.G = [np.zeros_like(self.X[0]) for _ in range(self.P)]
        self.f = [np.zeros_like(self.X[0]) for _ in range(self.P)]
        self.pstar = -1
        self.fmax = np.inf
        self.nsteps = 0

    def forces(self):
        """Evaluate movable images, tangents and NEB forces at the current X (no update)."""
        P = self.P
        E, G = self.eval_images(self.X[1:P - 1])
        self.E[1:P - 1] = E
        for p in range(1, P - 1):
            self.G[p] = G[p - 1]
        # climbing image: argmax over interior energies, lowest index on exact tie (O6)
        self.pstar = 1 + int(np.argmax(self.E[1:P - 1])) if self.climb else -1
        for p in range(1, P - 1):
            tau, tp, tm = improved_tangent(self.X[p - 1], self.X[p], self.X[p + 1], self.E[p - 1], self.E[p], self.E[p + 1])
            self.f[p] = neb_force(self.G[p], tau, tp, tm, self.k, climbing=(p == self.pstar))
        # O8: fmax over movable images and rows
        self.fmax = max(float(np.max(np.sqrt(np.sum(self.f[p] ** 2, axis=1)))) for p in range(1, P - 1))
        return self.f

    def step(self):
        """One NEB iteration: forces at X, then one FIRE update of all movable images."""
        P = self.P
        self.forces()
        f = np.stack(self.f[1:P - 1])
        rows = self.X[0].shape[0]
        delta = self.fire.step(f, (P - 2) * rows)
        for p in range(1, P - 1):
            x = self.X[p] + delta[p - 1]
            self.X[p] = self.post_update(x) if self.post_update else x
        self.nsteps += 1
        return self.fmax

    def run(self, fmax_tol, max_steps):
        for _ in range(max_steps):
            if self.step() < fmax_tol:
                break
        return self.fmax

    @property
    def barrier(self):
        """O8: E_{p*} - E_0 (highest interior energy if no climbing image)."""
        p = self.pstar if self.pstar > 0 else 1 + int(np.argmax(self.E[1:self.P - 1]))
        return self.E[p] - self.E[0]

    def segment_lengths(self):
        """O8: d_p = |X_{p+1} - X_p|, p = 0..P-2."""
        return np.array([np.sqrt(np.sum((self.X[p + 1] - self.X[p]) ** 2)) for p in range(self.P - 1)])
