"""The crystal band of CFNEB -- CPU ORACLE, TEST INFRASTRUCTURE ONLY.

One `step()` = one CFNEB iteration in the order of PAPER.md "IMPLEMENTATION": map each image
to generalized coordinates via the cell filter -> force evaluation -> NEB iteration (-> adjust the
image distribution, `adapt()`).  Composition of O0-O9:

  O0 input mapping          cellfilter.input_mapping        Eq. 10, 15
  O1 cell map D = sqrt(B)   cellfilter.cell_map
  O2 neighbours             forcefield.c
  O3 U, F, V                forcefield.c                    Eq. 4, 5, 8
  O4 generalized force      cellfilter.generalized_force    Eq. 17
  O5-O8                     neb.py                          Eq. 1, refs [12], [13]
  O9 adaptive control       adapt() below                   P:128 (reading A16; hand-worked pin)

External pressure (reading A25; the paper's graphite band is "under 40GPa", Fig. 3 caption, without
equations): a hydrostatic pressure p replaces U by the enthalpy H = U + p Omega, Omega = |det h|.  With the
right-multiplication strain of Eq. 2, Omega(eps) = Omega det(I + eps), so by Eq. 3 the virial of H is
V - p Omega I; H is the energy the tangent (O5), the climbing image (O6) and the barrier (O8) see.
"""
import numpy as np

from . import cellfilter as cf
from . import forcefield as ff
from .neb import Band, Fire


def auto_cell_factor(h0, n_atoms):
    """A13: lam = Omega0^(1/3) N^(1/6) (the Jacobian of ref [5]); lam = 1 is the paper literally."""
    return abs(np.linalg.det(h0)) ** (1.0 / 3.0) * n_atoms ** (1.0 / 6.0)


class CrystalEvaluator:
    """Callback for neb.Band: X = [R~ ; lam*B] -> (E, G) through O1-O4."""

    def __init__(self, h0, potential, pot, r_list, max_neighbors, lam=1.0, cell_mode=cf.CELL_B, brute=False,
                 threads=None, pressure=0.0, types=None):
        self.h0 = np.array(h0, dtype=np.float64)
        self.potential = int(potential)
        self.pot = np.array(pot, dtype=np.float64)
        self.r_list = float(r_list)
        self.cap = int(max_neighbors)
        self.lam = float(lam)
        self.cell_mode = cell_mode
        self.brute = brute
        self.threads = threads
        self.pressure = float(pressure)
        self.types = None if types is None else np.ascontiguousarray(types, dtype=np.int32)  # NEP-shaped potential only
        self.last = None  # (F, V, D, h) of the last evaluation, for parity hooks

    def deformation(self, X):
        Rt, C = cf.unpack(X, self.lam)
        D = C if self.cell_mode == cf.CELL_D else cf.cell_map(C)
        return Rt, D

    def __call__(self, X_list):
        Rts, Ds, hs = [], [], []
        for X in X_list:
            Rt, D = self.deformation(X)
            Rts.append(Rt)
            Ds.append(D)
            hs.append(self.h0 @ D)  # h = h0 D
        ff.set_types(self.types)
        E, F, V = ff.eval_images(np.stack(Rts), self.h0, np.stack(hs), self.potential, self.pot, self.r_list,
                                 self.cap, brute=self.brute, threads=self.threads)
        if self.pressure != 0.0:  # A25: H = U + p Omega;  V_H = V - p Omega I  (Eq. 2-3)
            E = np.array(E, dtype=np.float64)
            V = np.array(V, dtype=np.float64)
            for q in range(len(X_list)):
                omega = abs(np.linalg.det(hs[q]))
                E[q] += self.pressure * omega
                V[q] -= self.pressure * omega * np.eye(3)
        G = [cf.generalized_force(F[q], V[q], Ds[q], self.lam, self.cell_mode) for q in range(len(X_list))]
        self.last = dict(F=F, V=V, D=np.stack(Ds), h=np.stack(hs))
        return list(E), G


class CFNEB:
    """Cell-filter NEB band.  pos[P,N,3] Cartesian, cells[P,3,3] (rows = lattice vectors)."""

    def __init__(self, pos, cells, potential, pot, r_cut, k_spring=1.0, climb=True, cell_mode=cf.CELL_B,
                 cell_factor=1.0, fire=None, skin=0.3, max_neighbors=128, brute=False, threads=None, pressure=0.0,
                 types=None):
        pos = np.asarray(pos, dtype=np.float64)
        cells = np.asarray(cells, dtype=np.float64)
        self.N = pos.shape[1]
        self.h0 = cells[0].copy()  # A7: reference cell = cell of the initial endpoint
        self.lam = auto_cell_factor(self.h0, self.N) if cell_factor == 0 else float(cell_factor)
        self.cell_mode = cell_mode
        self.fire_params = dict(fire or {})
        X = []
        for p in range(pos.shape[0]):
            Rt, B, D = cf.input_mapping(pos[p], cells[p], self.h0)
            X.append(cf.pack(Rt, D if cell_mode == cf.CELL_D else B, self.lam))
        self.evaluator = CrystalEvaluator(self.h0, potential, pot, r_cut + skin, max_neighbors, self.lam, cell_mode,
                                          brute, threads, pressure, types)
        self.band = Band(X, self.evaluator, k_spring=k_spring, climb=climb, fire=self.fire_params,
                         post_update=self._post_update)

    def _post_update(self, X):
        if self.cell_mode == cf.CELL_B:  # O7 step 4: B <- 1/2 (B + B^T)
            X = X.copy()
            X[-3:] = 0.5 * (X[-3:] + X[-3:].T)
        elif self.cell_mode == cf.CELL_FIXED:
            pass
        return X

    # -- the hot path -------------------------------------------------------------------------
    def step(self, n=1):
        for _ in range(n):
            self.band.step()
        return self.band.fmax

    def run(self, fmax_tol, max_steps):
        return self.band.run(fmax_tol, max_steps)

    # -- views ---------------------------------------------------------------------------------
    @property
    def P(self):
        return self.band.P

    def get_path(self):
        """Cartesian positions R = R~ D, cells h = h0 D (rotation-free: D = sqrt(B)), energies."""
        pos, cells = [], []
        for X in self.band.X:
            Rt, D = self.evaluator.deformation(X)
            pos.append(Rt @ D)
            cells.append(self.h0 @ D)
        return np.stack(pos), np.stack(cells), self.band.E.copy()

    def get_state(self):
        """Generalized coordinates X[P,N+3,3] and FIRE velocities v[P,N+3,3] (zero rows for endpoints)."""
        X = np.stack(self.band.X)
        v = np.zeros_like(X)
        v[1:-1] = self.band.fire.v
        return X, v

    # -- O9: adaptive image control (reading A16) -----------------------------------------
    def adapt(self, d_insert, d_delete):
        """At most one deletion and one insertion per call.  Returns (n_inserted, n_deleted)."""
        b = self.band
        n_ins = n_del = 0
        d = b.segment_lengths()
        # (i) delete the interior, non-climbing image q minimising d_{q-1} + d_q, if below d_delete, P > 3
        if b.P > 3:
            cand = [(d[q - 1] + d[q], q) for q in range(1, b.P - 1) if q != b.pstar]
            if cand:
                s, q = min(cand)
                if s < d_delete:
                    self._delete(q)
                    n_del = 1
                    d = b.segment_lengths()
        # (ii) insert at the midpoint of the longest segment if above d_insert
        q = int(np.argmax(d))
        if d[q] > d_insert and (self.max_images is None or b.P < self.max_images):
            self._insert(q)
            n_ins = 1
        if n_ins or n_del:
            self._reset_fire()
        return n_ins, n_del

    max_images = None

    def insert_image(self, after):
        self._insert(after)
        self._reset_fire()

    def delete_image(self, index):
        self._delete(index)
        self._reset_fire()

    def _insert(self, q):
        b = self.band
        Xn = 0.5 * (b.X[q] + b.X[q + 1])
        b.X.insert(q + 1, Xn)
        b.E = np.insert(b.E, q + 1, np.nan)  # evaluated on the next step
        b.G.insert(q + 1, np.zeros_like(Xn))
        b.f.insert(q + 1, np.zeros_like(Xn))
        if b.pstar > q:
            b.pstar += 1
        b.P += 1

    def _delete(self, q):
        b = self.band
        del b.X[q], b.G[q], b.f[q]
        b.E = np.delete(b.E, q)
        if b.pstar > q:
            b.pstar -= 1
        b.P -= 1

    # -- O10: arc-length re-parametrisation ("the image distribution is automatically adjusted ... based on
    #    local spacing in configuration space"; reading A27) -------------------------------
    def reparametrize(self, hold_climbing=True):
        """Redistribute the interior images at equal arc length along the band's own polyline in X.

        With s_p = sum_{q<p} |X_{q+1} - X_q| and L = s_{P-1}, image p moves to the point of the polyline at arc length
        p L / (P-1): X_q + t (X_{q+1} - X_q) on the segment q that contains it.  hold_climbing: the climbing image
        stays where it is and each side of it is redistributed on its own with its own number of images (the
        saddle estimate is not smeared).  Endpoints never move.  FIRE restarts as after any O9 change."""
        b = self.band
        old = [x.copy() for x in b.X]
        d = b.segment_lengths()
        s = np.concatenate([[0.0], np.cumsum(d)])
        knots = [0, b.P - 1]
        if hold_climbing and 0 < b.pstar < b.P - 1:
            knots = [0, b.pstar, b.P - 1]
        for lo, hi in zip(knots[:-1], knots[1:]):
            for p in range(lo + 1, hi):
                target = s[lo] + (s[hi] - s[lo]) * (p - lo) / (hi - lo)
                q = lo
                while q < hi - 1 and s[q + 1] <= target:   # segment q with s_q <= target < s_{q+1}
                    q += 1
                t = (target - s[q]) / (s[q + 1] - s[q]) if s[q + 1] > s[q] else 0.0
                x = old[q] + t * (old[q + 1] - old[q])
                b.X[p] = self._post_update(x) if hasattr(self, "cell_mode") else x
                b.E[p] = np.nan  # evaluated on the next step
        self._reset_fire()

    def _reset_fire(self):
        b = self.band
        b.fire = Fire((b.P - 2,) + b.X[0].shape, **self.fire_params)


def relax_endpoint(R, h, potential, pot, r_cut, fmax_tol=1e-4, max_steps=20000, cell_factor=0.0, fire=None,
                   skin=0.3, max_neighbors=128, cell_mode=cf.CELL_B, pressure=0.0, h_ref=None, types=None):
    """Cell-filter FIRE relaxation of one structure (BASELINE.json configs: "both endpoints cell-relaxed").

    Same generalized coordinates and forces as the band (O0-O4, O7) with f = G (no NEB projection).
    h_ref: reference cell h0 of the generalized coordinates ("a reference cell", A7); default the structure's
    own cell.  A band relaxes its final endpoint in the frame of its initial endpoint's cell.
    Returns (R, h, E, fmax, n_steps).
    """
    R = np.asarray(R, dtype=np.float64)
    h = np.asarray(h, dtype=np.float64)
    h0 = h if h_ref is None else np.asarray(h_ref, dtype=np.float64)
    N = R.shape[0]
    lam = auto_cell_factor(h0, N) if cell_factor == 0 else float(cell_factor)
    ev = CrystalEvaluator(h0, potential, pot, r_cut + skin, max_neighbors, lam, cell_mode, pressure=pressure, types=types)
    Rt, B, D = cf.input_mapping(R, h, h0)
    X = cf.pack(Rt, D if cell_mode == cf.CELL_D else B, lam)  # Eq. 14 coordinates (R~, D) / Eq. 17 (R~, B)
    fire = Fire((1,) + X.shape, **(fire or {}))
    E, fmax, it = np.nan, np.inf, 0
    for it in range(max_steps):
        Es, Gs = ev([X])
        E, G = Es[0], Gs[0]
        fmax = float(np.max(np.sqrt(np.sum(G * G, axis=1))))
        if fmax < fmax_tol:
            break
        X = X + fire.step(G[None], X.shape[0])[0]
        if cell_mode == cf.CELL_B:  # O7 step 4: B <- 1/2 (B + B^T); D of Eq. 14 is not symmetric in general
            X[-3:] = 0.5 * (X[-3:] + X[-3:].T)
    Rt, D = ev.deformation(X)
    return Rt @ D, h0 @ D, E, fmax, it
