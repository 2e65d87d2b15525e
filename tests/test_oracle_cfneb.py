"""Pins for oracle/cfneb.py (the crystal band): the vacancy-hop barrier of BASELINE.json configs[0] against
an independent constrained relaxation, rotation-freeness of the band, the stored lattice
constants, the adaptive control (O9: structural invariants, and a hand-worked band whose expected deletion,
insertion and resulting order are written out from the rule of reading A16), and the one-pass reduction algebra
of SURVEY.md §8(d)."""
import numpy as np
import pytest

from cfneb_workloads import (CONFIGS, bain_endpoints, bcc_supercell, fcc_supercell, linear_path,
                             load_lattice_constants, vacancy_endpoints_unrelaxed)
from oracle import cellfilter as cf
from oracle import cfneb as oc
from oracle import forcefield as ff
from oracle.neb import Fire, improved_tangent, neb_force


@pytest.fixture(scope="module")
def c0():
    spec = CONFIGS[0]
    a = load_lattice_constants()["lj_fcc_a"]
    fi, cell, ffin, _ = vacancy_endpoints_unrelaxed(2, a)
    R0, h0, E0, fm0, _ = oc.relax_endpoint(fi @ cell, cell, 0, spec.pot, 2.5, fmax_tol=1e-7, fire=spec.fire)
    R1, h1, E1, fm1, _ = oc.relax_endpoint(ffin @ cell, cell, 0, spec.pot, 2.5, fmax_tol=1e-7, fire=spec.fire)
    assert fm0 < 1e-7 and fm1 < 1e-7
    pos, cells = linear_path(R0 @ np.linalg.inv(h0), h0, R1 @ np.linalg.inv(h1), h1, spec.n_images, spec.seed,
                             spec.noise_sigma)
    return dict(spec=spec, R0=R0, h0=h0, E0=E0, R1=R1, h1=h1, E1=E1, pos=pos, cells=cells)


def test_stored_lattice_constants_are_stress_free():
    lc = load_lattice_constants()
    frac, cell = fcc_supercell(2, 2, 2, lc["lj_fcc_a"])
    nb = ff.neighbors(frac @ cell, cell, cell, 2.5, 128)
    E, F, V = ff.energy_force_virial(frac @ cell, cell, cell, 0, CONFIGS[0].pot, nb)
    assert abs(np.trace(V)) < 1e-9 * 32 and abs(E / 32 - lc["lj_fcc_e_coh"]) < 1e-12
    fr, c0_, fr1, c1_ = bain_endpoints((3, 3, 3), lc["fs_bcc_a"], lc["fs_fcc_volume_ratio"])
    for frac, cell, nn in ((fr, c0_, 112), (fr1, c1_, 86)):
        nb = ff.neighbors(frac @ cell, cell, cell, 5.0, 256)
        E, F, V = ff.energy_force_virial(frac @ cell, cell, cell, 1, CONFIGS[2].pot, nb)
        assert np.all(nb[0] == nn)
        assert np.abs(V).max() < 1e-8 * len(frac) and np.abs(F).max() < 1e-10
    assert abs(np.linalg.det(c1_) / np.linalg.det(c0_) - lc["fs_fcc_volume_ratio"]) < 1e-12
    assert abs(c1_[2, 2] / c1_[0, 0] - np.sqrt(2.0)) < 1e-12  # c/a = sqrt 2


def test_c0_endpoints_equivalent_and_barrier_equals_constrained_saddle(c0):
    spec = c0["spec"]
    assert abs(c0["E0"] - c0["E1"]) < 1e-10  # symmetric hop
    neb = oc.CFNEB(c0["pos"], c0["cells"], 0, spec.pot, 2.5, k_spring=spec.k_spring, climb=True, cell_factor=0.0,
                   fire=spec.fire)
    neb.run(1e-5, 5000)
    assert neb.band.fmax < 1e-5 and neb.band.pstar == 3
    # independent route: symmetric path => saddle at the midpoint; minimise E with the hop coordinate of the
    # hopping atom fixed at the midpoint and the centre of mass of the others fixed; rest + cell relaxed.
    href = c0["h0"]
    lam = oc.auto_cell_factor(href, 31)
    ev = oc.CrystalEvaluator(href, 0, spec.pot, 2.8, 128, lam)
    Rt0, B0, _ = cf.input_mapping(c0["R0"], c0["h0"], href)
    Rt1, B1, _ = cf.input_mapping(c0["R1"], c0["h1"], href)
    X = cf.pack(0.5 * (Rt0 + Rt1), 0.5 * (B0 + B1), lam)
    u = Rt1[0] - Rt0[0]
    u /= np.linalg.norm(u)
    fire = Fire((1,) + X.shape, **spec.fire)
    for _ in range(5000):
        Es, Gs = ev([X])
        G = Gs[0].copy()
        G[0] -= np.dot(G[0], u) * u
        G[1:-3] -= G[1:-3].mean(axis=0)
        if np.max(np.sqrt((G * G).sum(axis=1))) < 1e-7:
            break
        X = X + fire.step(G[None], X.shape[0])[0]
        X[-3:] = 0.5 * (X[-3:] + X[-3:].T)
    assert np.abs(Gs[0]).max() < 1e-6  # the constrained minimum is a true stationary point
    saddle = Es[0] - c0["E0"]
    assert abs(neb.band.barrier - saddle) < 1e-6
    assert 4.9 < saddle < 5.1
    # paper-literal lam = 1 reaches the same barrier (a constant on the cell block only rescales its mass, A9/A13)
    neb1 = oc.CFNEB(c0["pos"], c0["cells"], 0, spec.pot, 2.5, k_spring=spec.k_spring, climb=True, cell_factor=1.0,
                    fire=spec.fire)
    neb1.run(2e-3, 3000)
    assert abs(neb1.band.barrier - saddle) < 1e-6


def test_band_is_rotation_free(c0):
    # a final endpoint supplied with a rigid rotation gives the same path, energies and barrier
    spec = c0["spec"]
    rng = np.random.default_rng(1)
    Q, _ = np.linalg.qr(rng.standard_normal((3, 3)))
    if np.linalg.det(Q) < 0:
        Q[:, 0] *= -1
    pos, cells = c0["pos"].copy(), c0["cells"].copy()
    pos[-1], cells[-1] = pos[-1] @ Q, cells[-1] @ Q
    pos[2], cells[2] = pos[2] @ Q.T, cells[2] @ Q.T
    a = oc.CFNEB(c0["pos"], c0["cells"], 0, spec.pot, 2.5, cell_factor=1.0, fire=spec.fire)
    b = oc.CFNEB(pos, cells, 0, spec.pot, 2.5, cell_factor=1.0, fire=spec.fire)
    a.step(5)
    b.step(5)
    pa, ca, Ea = a.get_path()
    pb, cb, Eb = b.get_path()
    assert np.abs(pa - pb).max() < 1e-10 and np.abs(ca - cb).max() < 1e-10 and np.abs(Ea - Eb).max() < 1e-9
    assert np.allclose(cb[-1], c0["cells"][-1], atol=1e-10)  # get_path returns the un-rotated cell h0 sqrt(B)


def test_one_pass_reduction_algebra_matches_direct_evaluation(c0):
    # f = G + c1 tau+ + c2 tau-, so f.v, f.f follow from ten dot products.
    spec = c0["spec"]
    neb = oc.CFNEB(c0["pos"], c0["cells"], 0, spec.pot, 2.5, cell_factor=1.0, fire=spec.fire)
    neb.step(3)
    b = neb.band
    b.forces()
    v = b.fire.v
    for p in range(1, b.P - 1):
        X0, X1, X2 = b.X[p - 1], b.X[p], b.X[p + 1]
        G, vv_ = b.G[p], v[p - 1]
        tp, tm = X2 - X1, X1 - X0
        d = lambda x, y: float(np.sum(x * y))
        pp, mm, pm, Gp, Gm, GG, Gv, pv, mv = d(tp, tp), d(tm, tm), d(tp, tm), d(G, tp), d(G, tm), d(G, G), d(G, vv_), d(tp, vv_), d(tm, vv_)
        # tangent weights (a, b) from the energies, O5
        tau = improved_tangent(X0, X1, X2, b.E[p - 1], b.E[p], b.E[p + 1])[0]
        A = np.linalg.lstsq(np.stack([tp.ravel(), tm.ravel()], axis=1), tau.ravel(), rcond=None)[0]
        a_, b_ = A
        tt = a_ * a_ * pp + 2 * a_ * b_ * pm + b_ * b_ * mm
        Gt = a_ * Gp + b_ * Gm
        if p == b.pstar:
            gam = -2 * Gt / tt
        else:
            gam = -Gt / tt + spec.k_spring * (np.sqrt(pp) - np.sqrt(mm)) / np.sqrt(tt)
        c1, c2 = gam * a_, gam * b_
        f = b.f[p]
        assert np.abs(f - (G + c1 * tp + c2 * tm)).max() < 1e-12 * np.abs(f).max() + 1e-13
        ff_ = GG + 2 * c1 * Gp + 2 * c2 * Gm + c1 * c1 * pp + 2 * c1 * c2 * pm + c2 * c2 * mm
        fv = Gv + c1 * pv + c2 * mv
        assert abs(ff_ - d(f, f)) < 1e-10 * d(f, f) and abs(fv - d(f, vv_)) < 1e-10 * max(abs(d(f, vv_)), 1e-3)


def test_get_path_round_trip_and_state(c0):
    spec = c0["spec"]
    neb = oc.CFNEB(c0["pos"], c0["cells"], 0, spec.pot, 2.5, cell_factor=1.0, fire=spec.fire)
    pos, cells, E = neb.get_path()
    assert np.abs(pos - c0["pos"]).max() < 1e-12 and np.abs(cells - c0["cells"]).max() < 1e-12
    X, v = neb.get_state()
    assert X.shape == (7, 34, 3) and np.all(v == 0)
    assert np.allclose(X[0, -3:], np.eye(3))  # B = I at the reference image


def test_adaptive_control_structural_invariants(c0):
    spec = c0["spec"]
    neb = oc.CFNEB(c0["pos"], c0["cells"], 0, spec.pot, 2.5, cell_factor=1.0, fire=spec.fire)
    neb.max_images = 9
    neb.step(3)
    d = neb.band.segment_lengths()
    Xold = [x.copy() for x in neb.band.X]
    q = int(np.argmax(d))
    n_ins, n_del = neb.adapt(d_insert=0.9 * d.max(), d_delete=0.0)
    assert (n_ins, n_del) == (1, 0) and neb.P == 8
    assert np.array_equal(neb.band.X[q + 1], 0.5 * (Xold[q] + Xold[q + 1]))  # exact midpoint
    assert np.all(neb.band.fire.v == 0) and neb.band.fire.first and neb.band.fire.dt == spec.fire["dt0"]
    neb.step(2)  # new image gets evaluated
    assert np.all(np.isfinite(neb.band.E))
    # deletion: never an endpoint, never the climbing image; P changes by -1
    ps = neb.band.pstar
    Xc = neb.band.X[ps].copy()
    n_ins, n_del = neb.adapt(d_insert=1e9, d_delete=1e9)
    assert (n_ins, n_del) == (0, 1) and neb.P == 7
    assert np.array_equal(neb.band.X[neb.band.pstar], Xc)
    assert np.array_equal(neb.band.X[0], Xold[0]) and np.array_equal(neb.band.X[-1], Xold[-1])
    # thresholds respected: nothing happens between them; max_images respected
    assert neb.adapt(d_insert=1e9, d_delete=0.0) == (0, 0)
    neb.max_images = 7
    assert neb.adapt(d_insert=0.0, d_delete=0.0) == (0, 0)


def test_relax_endpoint_in_every_cell_mode():
    """relax_endpoint in the Eq. 14 coordinates (R~, D) must stop at the same crystal as in the Eq. 17 coordinates
    (R~, B) -- the minimum does not depend on the coordinates it is searched in -- and with the cell fixed it must not
    move the cell while still lowering the energy (the pin of the CELL_D / CELL_FIXED branches)."""
    spec = CONFIGS[0]
    f0, cell, _, _ = vacancy_endpoints_unrelaxed(2, 1.60)   # off the stress-free lattice constant
    kw = dict(fmax_tol=1e-8, max_steps=6000, cell_factor=0.0, fire=spec.fire)
    out = {m: oc.relax_endpoint(f0 @ cell, cell, 0, spec.pot, 2.5, cell_mode=m, **kw) for m in (cf.CELL_B, cf.CELL_D, cf.CELL_FIXED)}
    (Rb, hb, Eb, fb, _), (Rd, hd, Ed, fd, _), (Rf, hf, Ef, ff_, _) = out[cf.CELL_B], out[cf.CELL_D], out[cf.CELL_FIXED]
    assert fb < 1e-8 and fd < 1e-8 and ff_ < 1e-8
    assert abs(Eb - Ed) < 1e-10 and abs(np.linalg.det(hb) - np.linalg.det(hd)) < 1e-6
    assert np.abs(hd - hd.T).max() < 1e-7        # no torque on a cubic cell: D stays symmetric although Eq. 14 does not force it
    assert np.array_equal(hf, cell) and Eb < Ef - 1.0
    nb = ff.neighbors(f0 @ cell, cell, cell, 2.5, 128)
    E_start = ff.energy_force_virial(f0 @ cell, cell, cell, 0, spec.pot, nb)[0]
    assert Ef < E_start - 1e-3                   # the atoms around the vacancy relaxed


def _line_band(xs, pstar):
    """A band of 1-row, 1-column images at the given abscissae (no crystal behind it): only what adapt() touches."""
    from oracle.neb import Band
    neb = object.__new__(oc.CFNEB)
    neb.fire_params = {}
    neb.band = Band([np.array([[x]]) for x in xs], lambda Xs: ([0.0] * len(Xs), [np.zeros((1, 1)) for _ in Xs]))
    neb.band.pstar = pstar
    return neb


def _abscissae(neb):
    return [float(x[0, 0]) for x in neb.band.X]


def test_adaptive_control_hand_worked_band():
    """Pin of O9 ("inserting or removing replicas based on local spacing in configuration space"; rule = reading
    A16).  Every expected index and order below is worked out by hand from the rule's text,
    not by oracle code.

    Six images on a line at x = 0, 1, 1.2, 1.5, 3.5, 4.5: segment lengths d = 1, 0.2, 0.3, 2, 1.
    Rule (i): delete the interior, non-climbing image q minimising d_{q-1} + d_q if that sum < d_delete:
        q = 1: 1 + 0.2 = 1.2;  q = 2: 0.2 + 0.3 = 0.5;  q = 3: 0.3 + 2 = 2.3;  q = 4: 2 + 1 = 3.
    Rule (ii), on the band after (i): insert the midpoint of the longest segment if it is longer than d_insert."""
    xs = [0.0, 1.0, 1.2, 1.5, 3.5, 4.5]
    # climbing image 4 (x = 3.5): the minimum 0.5 belongs to image 2 (x = 1.2) -> deleted.  Then d = 1, 0.5, 2, 1:
    # segment 2 (1.5 -> 3.5) is the longest -> midpoint 2.5 inserted after image 2.  The climbing image keeps x = 3.5:
    # index 4 -> 3 (deletion below it) -> 4 (insertion below it).
    neb = _line_band(xs, pstar=4)
    assert neb.adapt(d_insert=1.5, d_delete=0.6) == (1, 1)
    assert _abscissae(neb) == [0.0, 1.0, 1.5, 2.5, 3.5, 4.5] and neb.band.pstar == 4 and neb.P == 6
    assert neb.band.fire.first and np.all(neb.band.fire.v == 0) and neb.band.fire.v.shape[0] == 4  # FIRE restarted
    # the sum must be BELOW d_delete (0.5 is not < 0.5), the segment ABOVE d_insert (2 is not > 2)
    neb = _line_band(xs, pstar=4)
    assert neb.adapt(d_insert=2.0, d_delete=0.5) == (0, 0) and _abscissae(neb) == xs
    # deletion only: the insertion test sees the band after the deletion (longest segment still 2)
    neb = _line_band(xs, pstar=4)
    assert neb.adapt(d_insert=2.5, d_delete=0.6) == (0, 1) and _abscissae(neb) == [0.0, 1.0, 1.5, 3.5, 4.5]
    assert neb.band.pstar == 3
    # the min-sum image IS the climbing image (p* = 2): it is never a candidate.  The smallest sum among the others
    # is q = 1 (1.2): not below d_delete = 1.0 -> nothing deleted although 0.5 < 1.0 ...
    neb = _line_band(xs, pstar=2)
    assert neb.adapt(d_insert=1e9, d_delete=1.0) == (0, 0) and _abscissae(neb) == xs and neb.band.pstar == 2
    # ... and with d_delete = 1.3 image 1 (x = 1) goes, the climbing image moves from index 2 to 1, x = 1.2 kept
    neb = _line_band(xs, pstar=2)
    assert neb.adapt(d_insert=1e9, d_delete=1.3) == (0, 1) and _abscissae(neb) == [0.0, 1.2, 1.5, 3.5, 4.5]
    assert neb.band.pstar == 1
    # insertion below the climbing image shifts it up; insertion above does not.  d = 1, 0.2, 0.3, 2, 1 -> segment 3
    neb = _line_band(xs, pstar=4)
    assert neb.adapt(d_insert=1.9, d_delete=0.0) == (1, 0) and _abscissae(neb) == [0.0, 1.0, 1.2, 1.5, 2.5, 3.5, 4.5]
    assert neb.band.pstar == 5
    neb = _line_band(xs, pstar=1)
    assert neb.adapt(d_insert=1.9, d_delete=0.0) == (1, 0) and neb.band.pstar == 1
    # ties go to the lowest index (A16): equispaced band 0..4 with p* = 2 -> sums all 2 -> image 1 deleted; then
    # d = 2, 1, 1 -> segment 0 inserted at x = 1 again.  max_images caps the insertion, P > 3 the deletion.
    neb = _line_band([0.0, 1.0, 2.0, 3.0, 4.0], pstar=2)
    assert neb.adapt(d_insert=1e9, d_delete=2.5) == (0, 1) and _abscissae(neb) == [0.0, 2.0, 3.0, 4.0]
    neb = _line_band([0.0, 1.0, 2.0, 3.0, 4.0], pstar=3)
    assert neb.adapt(d_insert=0.5, d_delete=0.0) == (1, 0) and _abscissae(neb) == [0.0, 0.5, 1.0, 2.0, 3.0, 4.0]
    neb = _line_band([0.0, 1.0, 2.0, 3.0, 4.0], pstar=3)
    neb.max_images = 5
    assert neb.adapt(d_insert=0.5, d_delete=0.0) == (0, 0)
    neb = _line_band([0.0, 1.0, 2.0], pstar=-1)
    assert neb.adapt(d_insert=1e9, d_delete=1e9) == (0, 0)   # P = 3: the last interior image stays


def _plane_band(pts, pstar):
    from oracle.neb import Band
    neb = object.__new__(oc.CFNEB)
    neb.fire_params = {}
    neb.band = Band([np.array([p], dtype=float) for p in pts], lambda Xs: ([0.0] * len(Xs), [np.zeros((1, 2)) for _ in Xs]))
    neb.band.pstar = pstar
    return neb


def test_reparametrize_equal_arc_length():
    """Pin of the arc-length re-parametrisation (reading A27 of P:128): hand-worked polylines, the straight-line case
    (equal chords to 1e-12), identity on an equispaced band, every new image on the old polyline at arc length
    p L / (P - 1), endpoints untouched, the climbing image held."""
    pts = lambda neb: [tuple(float(c) for c in x[0]) for x in neb.band.X]
    # L-shaped polyline (0,0) -> (1,0) -> (1,3), bunched images: length 4, five images -> arc lengths 1, 2, 3
    neb = _plane_band([(0, 0), (0.25, 0), (0.5, 0), (1, 0), (1, 3)], pstar=-1)
    neb.reparametrize(hold_climbing=True)
    assert pts(neb) == [(0.0, 0.0), (1.0, 0.0), (1.0, 1.0), (1.0, 2.0), (1.0, 3.0)]
    assert neb.band.fire.first and np.all(neb.band.fire.v == 0) and np.all(np.isnan(neb.band.E[1:-1]))
    # the same band with the climbing image (index 3, the corner) held: two images share the first leg of length 1,
    # none lies on the second
    neb = _plane_band([(0, 0), (0.25, 0), (0.5, 0), (1, 0), (1, 3)], pstar=3)
    neb.reparametrize(hold_climbing=True)
    assert np.allclose(np.array(pts(neb)), [(0, 0), (1 / 3, 0), (2 / 3, 0), (1, 0), (1, 3)], atol=1e-15)
    neb = _plane_band([(0, 0), (0.25, 0), (0.5, 0), (1, 0), (1, 3)], pstar=3)
    neb.reparametrize(hold_climbing=False)
    assert pts(neb) == [(0.0, 0.0), (1.0, 0.0), (1.0, 1.0), (1.0, 2.0), (1.0, 3.0)]
    # straight line, unequal spacing -> equal chords
    rng = np.random.default_rng(5)
    u = rng.standard_normal(2)
    ts = np.array([0.0, 0.03, 0.4, 0.45, 0.5, 0.97, 1.0])
    neb = _plane_band([tuple(t * u) for t in ts], pstar=-1)
    neb.reparametrize()
    dl = neb.band.segment_lengths()
    assert np.abs(dl - dl.mean()).max() < 1e-12 * dl.mean()
    # equispaced band: identity to round-off
    neb = _plane_band([tuple(t * u) for t in np.linspace(0, 1, 7)], pstar=-1)
    before = np.stack(neb.band.X)
    neb.reparametrize()
    assert np.abs(np.stack(neb.band.X) - before).max() < 1e-15
    # general polyline in the plane: every new image lies on the old polyline at arc length p L / (P - 1)
    old = rng.standard_normal((9, 2)).cumsum(axis=0)
    neb = _plane_band([tuple(p) for p in old], pstar=-1)
    neb.reparametrize()
    new = np.stack(neb.band.X)[:, 0]
    seg = np.linalg.norm(np.diff(old, axis=0), axis=1)
    s = np.concatenate([[0], np.cumsum(seg)])
    assert np.array_equal(new[0], old[0]) and np.array_equal(new[-1], old[-1])
    for p in range(1, 8):
        best = None
        for q in range(8):   # brute force: closest point of every old segment
            a, b_ = old[q], old[q + 1]
            t = np.clip(np.dot(new[p] - a, b_ - a) / np.dot(b_ - a, b_ - a), 0, 1)
            dist = np.linalg.norm(new[p] - (a + t * (b_ - a)))
            arc = s[q] + t * seg[q]
            if abs(arc - p * s[-1] / 8) < 1e-9:
                best = dist if best is None else min(best, dist)
        assert best is not None and best < 1e-12


def test_bain_band_barrier_equals_the_saddle_of_the_closed_form_surface():
    """Pin of the Bain bands (BASELINE.json configs[2-4]) and of the whole crystal machinery on the FS potential with
    cell degrees of freedom: CI-NEB in the cell-filter coordinates, run to fmax < 1e-6 on a 54-atom cell, must stop
    at the saddle of the two-variable lattice-sum surface E(a, c) (tests/bain_surface.py: no tangent, no projection,
    no cell filter, no optimizer in it).  Barrier per atom to 1e-9; the same number holds for any supercell."""
    from bain_surface import energy_per_atom, saddle
    from cfneb_workloads import build_workload
    spec, pos, cells = build_workload(2, 9, dims=(3, 3, 3))
    N = pos.shape[1]
    orc = oc.CFNEB(pos, cells, spec.potential, spec.pot, spec.r_cut, k_spring=spec.k_spring, climb=True, cell_factor=0.0,
                   fire=spec.fire, skin=spec.skin, max_neighbors=256)
    fmax = orc.run(1e-6, 8000)
    assert fmax < 1e-6
    P_, C_, E_ = orc.get_path()
    a_bcc = load_lattice_constants()["fs_bcc_a"]
    e_bcc = energy_per_atom(a_bcc, a_bcc, spec.pot)
    assert abs(E_[0] / N - e_bcc) < 1e-12                           # endpoint energy = the lattice sum
    h = C_[orc.band.pstar] / 3.0                                    # climbing image, per conventional cell
    assert np.abs(h - np.diag(np.diag(h))).max() < 1e-9 and abs(h[0, 0] - h[1, 1]) < 1e-9   # it stayed tetragonal
    a_s, c_s, e_s, eig = saddle(h[0, 0], h[2, 2], spec.pot)
    assert eig[0] < 0.0 < eig[1]                                     # first-order saddle of the surface
    assert 1.0 < c_s / a_s < np.sqrt(2.0)
    assert abs(orc.band.barrier / N - (e_s - e_bcc)) < 1e-9
    assert 0.12 < e_s - e_bcc < 0.13
