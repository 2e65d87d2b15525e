"""GPU parity: the CUDA path (through the C ABI, via the ctypes binding) against the CPU oracle on the same
seeded inputs.  Tolerances are BASELINE.json north_star's: neighbour lists bit-exact after sorting; per-atom
forces, energies and virials to relative 1e-10; one full NEB step to relative 1e-9; converged barrier to 1e-4.

"relative" for an array means max|a - b| <= tol * max|b| (the array's own scale): forces and virials of a
near-equilibrium crystal are sums of cancelling pair terms, so an element-wise relative error is undefined at
the zeros; DESIGN.md "Tolerances" derives this form.
"""
import numpy as np
import pytest

from cfneb_workloads import CONFIGS, build_workload

pytestmark = pytest.mark.gpu

TOL_FORCE = 1e-10
TOL_STEP = 1e-9


def rel(a, b):
    a, b = np.asarray(a), np.asarray(b)
    s = np.max(np.abs(b))
    return float(np.max(np.abs(a - b)) / (s if s > 0 else 1.0))


def record_branches(orc):
    """Instrument the ORACLE side of a parity pair: orc.branches collects which branch of the FIRE state machine (O7:
    first / uphill / grow / downhill / clip = the step-length limit A4 was active) and of the improved tangent (O5:
    up / down / ext+ / ext- / tie / flat) every oracle step takes, so that a test can assert the branches it claims to
    compare -- a quiet change of a workload cannot un-test one.  Nothing of the CUDA path is read."""
    orc.branches = set()
    fire = orc.band.fire
    inner = fire.step

    def fire_step(f, n_rows):
        if fire.first:
            orc.branches.add("first")
        elif np.sum(f * fire.v) > 0.0:
            orc.branches.add("uphill")
            if fire.n_pos > fire.nmin:
                orc.branches.add("grow")
        else:
            orc.branches.add("downhill")
        delta = inner(f, n_rows)
        if np.sqrt(np.sum((fire.dt * fire.v) ** 2)) > fire.maxstep * np.sqrt(n_rows):
            orc.branches.add("clip")
            orc.clipped_steps = getattr(orc, "clipped_steps", 0) + 1
        return delta

    fire.step = fire_step
    band = orc.band
    inner_forces = band.forces

    def forces():
        f = inner_forces()
        for p in range(1, band.P - 1):  # the energies the tangents of this evaluation were chosen from
            Em, E0, Ep = band.E[p - 1], band.E[p], band.E[p + 1]
            if Ep > E0 > Em:
                orc.branches.add("up")
            elif Ep < E0 < Em:
                orc.branches.add("down")
            elif Ep == E0 == Em:
                orc.branches.add("flat")
            else:
                orc.branches.add("ext+" if Ep > Em else "ext-" if Ep < Em else "tie")
        return f

    band.forces = forces
    return orc


def make_pair(k, cell_factor=1.0, cell_mode=1, climb=None, n_images=None, max_images=None, pressure=0.0, fire=None, **over):
    """(oracle band, GPU band) on configs[k] inputs; fire: overrides of the config's FIRE constants (both sides)."""
    import paper_2510_16721_b200 as cf
    from oracle import cfneb as oc
    spec, pos, cells = build_workload(k, n_images)
    if fire:
        import copy
        spec = copy.copy(spec)                      # CONFIGS[k] itself is shared between tests
        spec.fire = dict(spec.fire, **fire)
    climb = spec.climb if climb is None else climb
    orc = oc.CFNEB(pos, cells, spec.potential, spec.pot, spec.r_cut, k_spring=spec.k_spring, climb=climb,
                   cell_mode=cell_mode, cell_factor=cell_factor, fire=spec.fire, skin=spec.skin,
                   max_neighbors=spec.max_neighbors, pressure=pressure)
    prm = cf.params_for(spec, cell_factor=cell_factor, cell_mode=cell_mode, climb=int(climb), max_images=max_images,
                        pressure=float(pressure), **over)
    gpu = cf.CFNEB(pos, cells, prm)
    return spec, record_branches(orc), gpu


def first_step_exact(orc, gpu):
    """ONE full iteration on both sides from the current (identical) state: displacement and velocity to 1e-9
    (BASELINE.json north_star), before round-off is amplified by the dynamics.  Returns X before the step."""
    X0, _ = orc.get_state()
    orc.step(1)
    gpu.step(1)
    Xo, vo = orc.get_state()
    Xg, vg = gpu.get_state()
    assert rel(Xg - X0, Xo - X0) < TOL_STEP, rel(Xg - X0, Xo - X0)
    assert rel(vg, vo) < TOL_STEP, rel(vg, vo)
    return X0


def sorted_triples(count, lst, shift):
    out = []
    for i in range(len(count)):
        c = int(count[i])
        t = np.concatenate([np.full((c, 1), i), lst[i, :c, None], shift[i, :c]], axis=1)
        out.append(t)
    t = np.concatenate(out, axis=0)
    return t[np.lexsort(t.T[::-1])]


# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("k", [0, 1, 2])
def test_neighbor_lists_bit_exact_after_sorting(k):
    from oracle import forcefield as ff
    spec, orc, gpu = make_pair(k)
    ev = orc.evaluator
    r_list = spec.r_cut + spec.skin
    for image in sorted({0, 1, orc.P // 2, orc.P - 1}):
        Rt, D = ev.deformation(orc.band.X[image])
        h = orc.h0 @ D
        cnt, lst, sh = ff.neighbors(Rt, orc.h0, h, r_list, spec.max_neighbors, brute=(k == 0))
        # guard: no pair within 1e-9 of the list radius (membership would be rounding-dependent, A20/A24):
        # the oracle's own search at r_list (1 -+ 1e-9) finds the same neighbours
        c_lo = ff.neighbors(Rt, orc.h0, h, r_list * (1.0 - 1e-9), spec.max_neighbors, brute=(k == 0))[0]
        c_hi = ff.neighbors(Rt, orc.h0, h, r_list * (1.0 + 1e-9), spec.max_neighbors, brute=(k == 0))[0]
        assert np.array_equal(c_lo, cnt) and np.array_equal(c_hi, cnt), "a pair sits within 1e-9 of the list radius"
        gc, gl, gs = gpu.get_neighbors(image)
        assert np.array_equal(np.sort(gc), np.sort(cnt)) and np.array_equal(gc, cnt)
        a, b = sorted_triples(gc, gl, gs), sorted_triples(cnt, lst, sh)
        assert a.shape == b.shape and np.array_equal(a, b)
        # symmetry (i; j, n) <=> (j; i, -n)
        fl = a.copy()
        fl[:, [0, 1]] = fl[:, [1, 0]]
        fl[:, 2:] *= -1
        assert np.array_equal(fl[np.lexsort(fl.T[::-1])], a)
    gpu.close()


@pytest.mark.parametrize("k,lam", [(0, 1.0), (0, 0.0), (1, 1.0), (2, 1.0), (2, 0.0)])
def test_forces_energies_virials_and_neb_force(k, lam):
    spec, orc, gpu = make_pair(k, cell_factor=lam)
    f_or = orc.band.forces()
    last = orc.evaluator.last
    F, V, fneb, E = gpu.get_forces()
    P = orc.P
    assert rel(E, orc.band.E) < TOL_FORCE
    assert rel(E[1:-1] - E[0], orc.band.E[1:-1] - orc.band.E[0]) < 1e-8  # energy differences along the band
    assert rel(F[1:-1], last["F"]) < TOL_FORCE
    assert rel(V[1:-1], last["V"]) < TOL_FORCE
    for p in range(1, P - 1):
        assert rel(F[p], last["F"][p - 1]) < TOL_FORCE
        assert rel(fneb[p], f_or[p]) < TOL_STEP
    assert np.all(fneb[0] == 0) and np.all(fneb[-1] == 0)
    st = gpu.get_status()
    assert st.climb_index == orc.band.pstar
    assert abs(st.barrier - orc.band.barrier) < 1e-9 * max(1.0, abs(orc.band.E[0]))
    if lam == 0.0:
        from oracle.cfneb import auto_cell_factor
        assert abs(st.cell_factor - auto_cell_factor(orc.h0, orc.N)) < 1e-12 * st.cell_factor
    gpu.close()


@pytest.mark.parametrize("k,lam,nsteps", [(0, 1.0, 30), (0, 0.0, 30), (1, 0.0, 20), (2, 0.0, 12), (1, 1.0, 10)])
def test_neb_steps_match_oracle(k, lam, nsteps):
    """X and v after 1, 2, ... n full iterations (K0-K6) against the oracle's step()."""
    spec, orc, gpu = make_pair(k, cell_factor=lam)
    X0, _ = orc.get_state()
    Xg, vg = gpu.get_state()
    assert rel(Xg, X0) < 1e-14 and np.all(vg == 0)
    checks = sorted({1, 2, 3, nsteps // 2, nsteps})
    done = 0
    for n in checks:
        orc.step(n - done)
        gpu.step(n - done)
        done = n
        Xo, vo = orc.get_state()
        Xg, vg = gpu.get_state()
        dX = rel(Xg - X0, Xo - X0)  # the displacement, not the (much larger) coordinate, carries the step
        dv = rel(vg, vo)
        growth = 4.0 ** (n - 1) if n < 6 else 1e3  # round-off is amplified by later steps, not by the first
        assert dX < TOL_STEP * min(growth, 1e3), (n, dX)
        assert dv < TOL_STEP * min(growth, 1e3), (n, dv)
        st = gpu.get_status()
        assert st.steps == n and st.error == 0
        assert abs(st.fmax - orc.band.fmax) <= 1e-8 * orc.band.fmax
        assert abs(st.dt - orc.band.fire.dt) < 1e-15 and abs(st.alpha - orc.band.fire.alpha) < 1e-15
        assert st.n_pos == orc.band.fire.n_pos
    # the branches of O5 / O7 these trajectories compare (recorded on the oracle side); the step-length limit and the
    # equal-energy tangents are not among them: test_step_length_limit_follows_oracle, test_equal_energy_tangents_*
    want = {"first", "uphill", "downhill", "up", "ext+"}
    if k != 2:
        want |= {"down", "ext-"}
    if nsteps >= 20:
        want |= {"grow"}
    assert want <= orc.branches and "clip" not in orc.branches, sorted(orc.branches)
    gpu.close()


def test_first_step_is_exact_to_1e9():
    """The north-star number: ONE full NEB step to 1e-9 relative, every config the oracle finishes in seconds."""
    for k in (0, 1, 2):
        spec, orc, gpu = make_pair(k, cell_factor=0.0)
        X0, _ = orc.get_state()
        orc.step(1)
        gpu.step(1)
        Xo, vo = orc.get_state()
        Xg, vg = gpu.get_state()
        assert rel(Xg - X0, Xo - X0) < TOL_STEP and rel(vg, vo) < TOL_STEP
        assert rel(Xg, Xo) < 1e-13
        gpu.close()


@pytest.mark.parametrize("k,maxstep,pattern", [(0, 1e-4, "11111111"), (2, 1e-4, "11111111"), (0, 3e-3, "00111111"),
                                               (2, 6e-3, "00111000")])
def test_step_length_limit_follows_oracle(k, maxstep, pattern):
    """Reading A4 (O7 step 3): the band's displacement is limited to maxstep sqrt((P-2)(N+3)) in the 2-norm.  K5 takes the
    limit from its one-pass |v_new|^2 and K6 applies it as a factor on dt; the oracle clips the materialised Delta.
    With maxstep this small the limit is active -- asserted on the oracle's own numbers -- from the first iteration
    (pattern 1...) or from the third on, after two free ones (the switch-on inside a trajectory; on configs[2] a downhill
    restart at the sixth iteration switches it off again).  A wrong row count in K5's limit (N for N + 3, P for P - 2)
    changes the clipped step by percents."""
    spec, orc, gpu = make_pair(k, cell_factor=0.0, fire=dict(maxstep=maxstep))
    X0, _ = orc.get_state()
    for n in range(1, 9):
        Xb, _ = orc.get_state()
        clipped_before = getattr(orc, "clipped_steps", 0)
        orc.step(1)
        gpu.step(1)
        clipped = getattr(orc, "clipped_steps", 0) > clipped_before
        assert clipped == (pattern[n - 1] == "1"), (n, clipped)
        Xo, vo = orc.get_state()
        Xg, vg = gpu.get_state()
        if clipped:  # the oracle's step has exactly the limit's length
            assert abs(np.linalg.norm(Xo[1:-1] - Xb[1:-1]) / (maxstep * np.sqrt((orc.P - 2) * (orc.N + 3))) - 1.0) < 1e-6
        growth = 4.0 ** (n - 1) if n < 6 else 1e3
        assert rel(Xg - X0, Xo - X0) < TOL_STEP * min(growth, 1e3), (n, rel(Xg - X0, Xo - X0))
        assert rel(vg, vo) < TOL_STEP * min(growth, 1e3), (n, rel(vg, vo))
        st = gpu.get_status()
        assert abs(st.dt - orc.band.fire.dt) < 1e-15 and st.n_pos == orc.band.fire.n_pos and st.error == 0
    assert "clip" in orc.branches and "first" in orc.branches and "uphill" in orc.branches
    gpu.close()


@pytest.mark.parametrize("climb", [True, False])
def test_equal_energy_tangents_follow_oracle(climb):
    """The equal-energy branches of the improved tangent (O5; reading A26: three equal energies -> bisector; E_{p+1} =
    E_{p-1} -> the last branch) compared with the oracle, with energies that tie BITWISE on both sides by construction:
    in the Eq. 14 coordinates (CELL_D, lam = 1) an image with deformation D R, R a rotation by pi about a cell axis
    (two columns of D negated), has every pair vector r = ds h0 D R with two components negated exactly, hence the same
    r^2, the same lists in the same order and the same energy bit for bit as the image with D -- while being a
    different point of the band (the cell rows differ), so the tangents are not zero.  Images 1, 2, 3 and 5 are such
    copies of one structure (flat at p = 2, ties at p = 4 with image 4 between them).  The state is an INPUT built from
    the oracle's X; the ties are asserted on the oracle's own energies, then on the kernel's."""
    spec, orc, gpu = make_pair(0, cell_factor=1.0, cell_mode=2, climb=climb)
    X, _ = orc.get_state()
    assert X.shape[0] == 7
    Rx, Ry, Rz = np.array([1.0, -1.0, -1.0]), np.array([-1.0, 1.0, -1.0]), np.array([-1.0, -1.0, 1.0])
    for p, R in ((2, Rz), (3, Rx), (5, Ry)):
        X[p] = X[1]
        X[p, -3:, :] = X[1, -3:, :] * R          # columns of D negated: D R
    for p in range(1, 6):
        orc.band.X[p] = X[p].copy()
    gpu.set_state(X)
    f_or = orc.band.forces()
    Eo = orc.band.E
    assert Eo[1] == Eo[2] == Eo[3] == Eo[5] and Eo[4] != Eo[3]
    assert {"flat", "tie"} <= orc.branches, sorted(orc.branches)
    F, V, fneb, E = gpu.get_forces()
    assert E[1] == E[2] == E[3] == E[5] and E[4] != E[3]      # the kernel's K5 sees the ties as well
    assert rel(E, Eo) < TOL_FORCE
    for p in range(1, 6):
        assert rel(fneb[p], f_or[p]) < TOL_STEP, (p, rel(fneb[p], f_or[p]))
    assert gpu.get_status().climb_index == orc.band.pstar
    first_step_exact(orc, gpu)
    assert gpu.get_status().error == 0
    gpu.close()


def test_c0_converged_barrier_matches_oracle():
    spec, orc, gpu = make_pair(0, cell_factor=0.0)
    orc.run(1e-4, 3000)
    for _ in range(60):
        gpu.step(50)
        if gpu.get_status().fmax < 1e-4:
            break
    st = gpu.get_status()
    assert st.fmax < 1e-4 and st.error == 0
    assert st.climb_index == orc.band.pstar == 3
    assert abs(st.barrier - orc.band.barrier) < 1e-4
    assert 4.9 < st.barrier < 5.1
    pos, cells, E = gpu.get_path()
    assert abs(E[0] - E[-1]) < 1e-9  # symmetric hop
    gpu.close()


def test_c1_barrier_after_fixed_budget():
    spec, orc, gpu = make_pair(1, cell_factor=0.0)
    orc.run(1e-3, 1500)
    n = orc.band.nsteps
    gpu.step(n)
    st = gpu.get_status()
    assert st.steps == n
    assert abs(st.barrier - orc.band.barrier) < 1e-4
    assert st.fmax < 2e-3
    gpu.close()


@pytest.mark.parametrize("mode", [0, 2])
def test_cell_modes_fixed_and_D(mode):
    """CELL_FIXED (no cell force) and the Eq. 14 D-variant follow the oracle too."""
    spec, orc, gpu = make_pair(0, cell_factor=1.0, cell_mode=mode)
    Xg0, _ = gpu.get_state()
    X0 = first_step_exact(orc, gpu)
    orc.step(4)
    gpu.step(4)
    Xo, vo = orc.get_state()
    Xg, vg = gpu.get_state()
    assert rel(Xg - X0, Xo - X0) < 1e-7 and rel(vg, vo) < 1e-7
    if mode == 0:  # O4: G_cell = 0; the cell rows only see the (here ~1e-16) tangent between the endpoint cells
        assert np.max(np.abs(Xg[:, -3:] - Xg0[:, -3:])) < 1e-12 and np.max(np.abs(Xo[:, -3:] - X0[:, -3:])) < 1e-12
    gpu.close()


@pytest.mark.parametrize("k,mode,p_ext", [(0, 1, 0.7), (0, 2, 0.7), (2, 1, 0.25)])
def test_external_pressure_enthalpy_band(k, mode, p_ext):
    """Reading A25 ("under 40GPa"): H = U + p Omega and V - p Omega I, in both cell coordinates (Eq. 14, Eq. 17).
    0.25 eV/A^3 = 40 GPa for the Finnis-Sinclair band."""
    spec, orc, gpu = make_pair(k, cell_factor=0.0, cell_mode=mode, pressure=p_ext, n_images=5 if k == 2 else None)
    f_or = orc.band.forces()
    F, V, fneb, E = gpu.get_forces()
    assert rel(E, orc.band.E) < TOL_FORCE
    assert rel(V[1:-1], orc.evaluator.last["V"]) < TOL_FORCE
    assert rel(fneb[1:-1], np.stack(f_or[1:-1])) < TOL_STEP
    # the pressure term is a large part of what is being compared
    _, cells, _ = orc.get_path()
    assert p_ext * abs(np.linalg.det(cells[1])) > 0.05 * abs(orc.band.E[1] - p_ext * abs(np.linalg.det(cells[1])))
    X0 = first_step_exact(orc, gpu)
    orc.step(3)
    gpu.step(3)
    Xo, vo = orc.get_state()
    Xg, vg = gpu.get_state()
    assert rel(Xg - X0, Xo - X0) < 1e-7 and rel(vg, vo) < 1e-7
    st = gpu.get_status()
    assert st.error == 0 and abs(st.barrier - orc.band.barrier) < 1e-9 * max(1.0, abs(orc.band.barrier))
    gpu.close()


def test_no_climbing_image():
    spec, orc, gpu = make_pair(1, cell_factor=0.0, climb=False)
    X0, _ = orc.get_state()
    orc.step(3)
    gpu.step(3)
    Xo, _ = orc.get_state()
    Xg, _ = gpu.get_state()
    assert rel(Xg - X0, Xo - X0) < 1e-8
    assert gpu.get_status().climb_index == -1
    gpu.close()


def test_insert_delete_and_adapt_follow_oracle():
    spec, orc, gpu = make_pair(1, cell_factor=0.0, max_images=14)
    orc.max_images = 14
    orc.step(4)
    gpu.step(4)
    orc.insert_image(2)
    gpu.insert_image(2)
    assert gpu.P == orc.P == 10
    Xo, vo = orc.get_state()
    Xg, vg = gpu.get_state()
    assert rel(Xg, Xo) < 1e-12 and np.all(vg == 0)
    assert np.array_equal(Xg[3], 0.5 * (Xg[2] + Xg[4]))  # midpoint exact
    orc.step(3)
    gpu.step(3)
    Xo, vo = orc.get_state()
    Xg, vg = gpu.get_state()
    assert rel(Xg, Xo) < 1e-11 and rel(vg, vo) < 1e-7
    assert np.isfinite(gpu.get_path(positions=False)[2]).all()
    q = 7 if gpu.get_status().climb_index != 7 else 6
    orc.delete_image(q)
    gpu.delete_image(q)
    assert gpu.P == orc.P == 9
    orc.step(2)
    gpu.step(2)
    assert rel(gpu.get_state()[0], orc.get_state()[0]) < 1e-11
    d = gpu.get_segment_lengths()
    assert rel(d, orc.band.segment_lengths()) < 1e-10
    # adaptive control: thresholds that force one insertion, then one deletion
    di, dd = 0.9 * d.max(), 0.0
    assert gpu.adapt(di, dd) == orc.adapt(di, dd) == (1, 0)
    assert gpu.P == orc.P == 10
    d = gpu.get_segment_lengths()
    di, dd = 10 * d.max(), 1.01 * np.min(d[:-1] + d[1:]) + 1.0
    ro, rg = orc.adapt(di, dd), gpu.adapt(di, dd)
    assert ro == rg and rg[1] == 1
    assert rel(gpu.get_state()[0], orc.get_state()[0]) < 1e-11
    orc.step(2)
    gpu.step(2)
    assert rel(gpu.get_state()[0], orc.get_state()[0]) < 1e-10
    gpu.close()


@pytest.mark.parametrize("k,hold", [(1, True), (1, False), (2, True)])
def test_reparametrize_follows_oracle(k, hold):
    """cfneb_reparametrize (kernels on the stream, nothing read back) against oracle.reparametrize: a band whose images
    were bunched by hand goes to equal arc length along its own polyline; endpoints and the held climbing image do not
    move by a bit; the band then keeps stepping with the oracle (lists kept or rebuilt by the staleness bound)."""
    spec, orc, gpu = make_pair(k, cell_factor=0.0, n_images=9 if k == 2 else None)
    orc.step(4)
    gpu.step(4)
    # bunch the images: pull every interior image but the climbing one towards its lower neighbour
    ps = orc.band.pstar
    assert gpu.get_status().climb_index == ps
    pos, cells, _ = orc.get_path()
    for p in range(1, orc.P - 1):
        if p != ps and p % 2 == 1:
            pos[p] = 0.7 * pos[p] + 0.3 * pos[p - 1]
            cells[p] = 0.7 * cells[p] + 0.3 * cells[p - 1]
    from oracle import cfneb as oc
    orc2 = oc.CFNEB(pos, cells, spec.potential, spec.pot, spec.r_cut, k_spring=spec.k_spring, climb=spec.climb, cell_factor=0.0,
                    fire=spec.fire, skin=spec.skin, max_neighbors=spec.max_neighbors)
    gpu.set_path(pos, cells)
    orc2.step(1)
    gpu.step(1)
    assert gpu.get_status().climb_index == orc2.band.pstar
    Xb, _ = gpu.get_state()
    d_before = gpu.get_segment_lengths()
    assert d_before.max() > 1.3 * d_before.min()
    orc2.reparametrize(hold_climbing=hold)
    gpu.reparametrize(hold_climbing=hold)
    Xo, vo = orc2.get_state()
    Xg, vg = gpu.get_state()
    assert rel(Xg - Xb, Xo - Xb) < 1e-10 and np.all(vg == 0)
    assert np.array_equal(Xg[0], Xb[0]) and np.array_equal(Xg[-1], Xb[-1])
    pstar = orc2.band.pstar
    if hold:
        assert np.array_equal(Xg[pstar], Xb[pstar])
        for lo, hi in ((0, pstar), (pstar, orc2.P - 1)):   # equal arc length on each side, measured along the old polyline
            seg = np.array([np.linalg.norm(Xb[q + 1] - Xb[q]) for q in range(lo, hi)])
            assert abs(sum(np.linalg.norm(Xg[q + 1] - Xg[q]) for q in range(lo, hi)) - seg.sum()) < 1e-2 * seg.sum()
    d_after = gpu.get_segment_lengths()
    assert rel(d_after, orc2.band.segment_lengths()) < 1e-10
    if not hold:
        assert d_after.max() < 1.02 * d_after.min()          # the polyline is nearly straight: chords ~ arcs
    st = gpu.get_status()
    assert st.dt == spec.fire["dt0"] and st.n_pos == 0 and st.error == 0
    orc2.step(3)
    gpu.step(3)
    Xo2, _ = orc2.get_state()
    Xg2, _ = gpu.get_state()
    assert rel(Xg2 - Xg, Xo2 - Xo) < 1e-7
    assert np.all(np.isfinite(gpu.get_path(positions=False)[2])) and gpu.get_status().error == 0
    gpu.close()


def test_image_control_errors():
    import paper_2510_16721_b200 as cf
    spec, orc, gpu = make_pair(0)
    for bad in (-1, 6, 99):
        with pytest.raises(cf.CfnebError) as e:
            gpu.insert_image(bad)
        assert e.value.code == cf.binding.ERANGE
    with pytest.raises(cf.CfnebError):  # band full (max_images = 7)
        gpu.insert_image(1)
    for bad in (0, 6, 7):
        with pytest.raises(cf.CfnebError):
            gpu.delete_image(bad)
    gpu.step(1)
    with pytest.raises(cf.CfnebError):  # the climbing image may not be deleted
        gpu.delete_image(gpu.get_status().climb_index)
    gpu.close()


def test_create_errors_and_sticky_device_errors():
    import paper_2510_16721_b200 as cf
    spec, pos, cells = build_workload(0)
    with pytest.raises(cf.CfnebError) as e:  # neighbour capacity too small: sticky device error surfaces in create
        cf.CFNEB(pos, cells, cf.params_for(spec, max_neighbors=16))
    assert e.value.code == cf.binding.ENEIGH_OVERFLOW
    with pytest.raises(cf.CfnebError) as e:
        cf.CFNEB(pos[:2], cells[:2], cf.params_for(spec), n_images=2)
    assert e.value.code == cf.binding.EINVAL
    bad = cells.copy()
    bad[3] = 0.0
    with pytest.raises(cf.CfnebError) as e:
        cf.CFNEB(pos, bad, cf.params_for(spec))
    assert e.value.code == cf.binding.ECELL
    with pytest.raises(cf.CfnebError) as e:  # more images than capacity
        cf.CFNEB(pos, cells, cf.params_for(spec, max_images=5))
    assert e.value.code == cf.binding.ERANGE
    with pytest.raises(cf.CfnebError):  # identical interior images: zero tangent
        p2 = pos.copy()
        p2[:] = pos[0]
        c2 = cells.copy()
        c2[:] = cells[0]
        g = cf.CFNEB(p2, c2, cf.params_for(spec))
        g.step(1)
        g.get_state()


def test_endpoints_only_constructor_and_get_path_roundtrip():
    import paper_2510_16721_b200 as cf
    spec, pos, cells = build_workload(1)
    gpu = cf.CFNEB(pos[[0, -1]], cells[[0, -1]], cf.params_for(spec), n_images=9)
    p, c, E = gpu.get_path()
    assert p.shape == pos.shape and rel(p[0], pos[0]) < 1e-15 and rel(p[-1], pos[-1]) < 1e-14
    assert rel(c[0], cells[0]) < 1e-15 and rel(c[-1], cells[-1]) < 1e-14
    X, _ = gpu.get_state()
    for q in range(9):  # linear in the generalized coordinates
        assert rel(X[q], X[0] + q / 8.0 * (X[-1] - X[0])) < 1e-14
    # explicit-path constructor: get_path returns what went in (cells rotation-free: inputs here are symmetric D)
    g2 = cf.CFNEB(pos, cells, cf.params_for(spec))
    p2, c2, E2 = g2.get_path()
    assert rel(p2, pos) < 1e-14 and rel(c2, cells) < 1e-14
    # set_path round trip restarts from the same state
    X_before, _ = g2.get_state()
    E_before = g2.get_path(positions=False)[2]
    g2.step(3)
    assert not np.array_equal(g2.get_state()[0], X_before)
    g2.set_path(pos, cells)
    assert np.array_equal(g2.get_state()[0], X_before) and np.all(g2.get_state()[1] == 0)
    assert np.array_equal(g2.get_path(positions=False)[2], E_before)
    st = g2.get_status()
    assert st.dt == spec.fire["dt0"] and st.n_pos == 0
    gpu.close()
    g2.close()


def test_rotated_final_endpoint_gives_the_same_band():
    """P:110 / P:124: B = D D^T removes rigid rotations -- a final endpoint supplied rotated by Q changes nothing."""
    import paper_2510_16721_b200 as cf
    spec, pos, cells = build_workload(0)
    th = 0.3
    Q = np.array([[np.cos(th), -np.sin(th), 0], [np.sin(th), np.cos(th), 0], [0, 0, 1.0]])
    pos_r, cells_r = pos.copy(), cells.copy()
    pos_r[-1] = pos[-1] @ Q
    cells_r[-1] = cells[-1] @ Q
    a = cf.CFNEB(pos, cells, cf.params_for(spec, cell_factor=0.0))
    b = cf.CFNEB(pos_r, cells_r, cf.params_for(spec, cell_factor=0.0))
    a.step(25)
    b.step(25)
    Xa, _ = a.get_state()
    Xb, _ = b.get_state()
    assert rel(Xb, Xa) < 1e-10
    assert abs(a.get_status().barrier - b.get_status().barrier) < 1e-9
    pa, ca, _ = a.get_path()
    pb, cb, _ = b.get_path()
    assert rel(cb, ca) < 1e-10  # returned un-rotated (documented in include/cfneb.h)
    a.close()
    b.close()


def test_bitwise_repeatable():
    import paper_2510_16721_b200 as cf
    spec, pos, cells = build_workload(2)
    out = []
    for _ in range(2):
        g = cf.CFNEB(pos, cells, cf.params_for(spec, cell_factor=0.0))
        g.step(8)
        out.append(g.get_state())
        g.close()
    assert np.array_equal(out[0][0], out[1][0]) and np.array_equal(out[0][1], out[1][1])


@pytest.mark.parametrize("k,n_before,n_after,over", [(2, 25, 30, dict()), (1, 7, 12, dict(cell_mode=2)), (2, 13, 20, dict(rebuild_every=9))])
def test_checkpoint_resume_is_bit_exact(k, n_before, n_after, over):
    """cfneb_get_checkpoint -> cfneb_destroy -> cfneb_create -> cfneb_set_state continues the band bit for bit
    (SURVEY.md section 5 checkpoint row; "structural information is always kept and updated on GPU"): X, v, the
    FIRE scalars, and -- because the order of a list's entries fixes the summation order -- the coordinates each
    neighbour list was built at with its staleness accounting (incl. the count-down of rebuild_every)."""
    import paper_2510_16721_b200 as cf
    spec, pos, cells = build_workload(k)
    prm = cf.params_for(spec, cell_factor=0.0, **over)
    a = cf.CFNEB(pos, cells, prm)
    a.step(n_before)
    ck = a.get_checkpoint()
    st_ck = a.get_status()
    a.step(n_after)
    Xa, va = a.get_state()
    sa = a.get_status()
    a.close()
    assert ck["fire"].steps == n_before and ck["fire"].first == 0
    assert np.any(ck["X_list"] != ck["X"])                    # some list is older than the checkpoint
    b = cf.CFNEB(pos, cells, prm)                             # a new handle from the same inputs
    b.step(3)                                                 # ... in some other state
    b.set_state(ck["X"], ck["v"], ck["X_list"], ck["list_aux"], ck["fire"])
    Xb0, vb0 = b.get_state()
    assert np.array_equal(Xb0, ck["X"]) and np.array_equal(vb0, ck["v"])
    sb0 = b.get_status()
    assert (sb0.dt, sb0.alpha, sb0.n_pos, sb0.steps) == (st_ck.dt, st_ck.alpha, st_ck.n_pos, n_before)
    r0 = sb0.rebuilds
    b.step(n_after)
    Xb, vb = b.get_state()
    sb = b.get_status()
    assert np.array_equal(Xb, Xa) and np.array_equal(vb, va)
    assert (sb.dt, sb.alpha, sb.n_pos, sb.fmax, sb.barrier, sb.steps) == (sa.dt, sa.alpha, sa.n_pos, sa.fmax, sa.barrier, sa.steps)
    if over.get("rebuild_every"):
        assert sb.rebuilds > r0 and sa.rebuilds > st_ck.rebuilds   # both windows rebuilt lists, at the same iterations
    # without X_list the lists are fresh: same band to round-off, FIRE state still restored
    c = cf.CFNEB(pos, cells, prm)
    c.set_state(ck["X"], ck["v"], None, None, ck["fire"])
    c.step(n_after)
    Xc, vc = c.get_state()
    assert rel(Xc - ck["X"], Xa - ck["X"]) < 1e-9 and c.get_status().n_pos == sa.n_pos
    # no FIRE state: a restart from the stored coordinates (v = 0, dt = dt0, first step)
    c.set_state(ck["X"])
    assert np.all(c.get_state()[1] == 0) and c.get_status().dt == spec.fire["dt0"]
    with pytest.raises(cf.CfnebError):
        c.set_state(ck["X"], ck["v"], ck["X_list"], None, ck["fire"])   # X_list without its accounting
    b.close()
    c.close()


@pytest.mark.parametrize("k,n_blocks,over", [(2, 0, dict()), (2, 3, dict(rebuild_every=4)), (1, 1, dict(cell_mode=2)), (0, 7, dict())])
def test_step_hosted_is_bit_identical_to_the_resident_band(k, n_blocks, over):
    """cfneb_step_hosted -- the state lives in host memory, image blocks are evaluated while later blocks are still
    being uploaded -- gives, bit for bit, the states of the device-resident band (graph-launched cfneb_step), list
    rebuilds included, for any number of blocks."""
    import paper_2510_16721_b200 as cf
    spec, pos, cells = build_workload(k)
    prm = cf.params_for(spec, cell_factor=0.0, **over)
    a = cf.CFNEB(pos, cells, prm)
    b = cf.CFNEB(pos, cells, prm)
    a.step(3)
    b.step(3)
    ck = b.get_checkpoint()
    X, v, fire = np.ascontiguousarray(ck["X"]), np.ascontiguousarray(ck["v"]), ck["fire"]
    for it in range(9):
        a.step(1)
        b.step_hosted(X, v, fire, n_blocks)
        Xa, va = a.get_state()
        assert np.array_equal(X, Xa) and np.array_equal(v, va), it
        sa = a.get_status()
        assert (fire.dt, fire.alpha, fire.n_pos, fire.steps, fire.first) == (sa.dt, sa.alpha, sa.n_pos, sa.steps, 0)
    sb = b.get_status()
    assert sb.error == 0 and sb.fmax == sa.fmax and sb.barrier == sa.barrier
    assert sb.rebuilds >= sa.rebuilds   # (the hosted step keeps the two endpoint lists up as well: rebuild_every counts for them too)
    with pytest.raises(cf.CfnebError):
        bad = cf.FireState(dt=-1.0, alpha=0.1, steps=0, n_pos=0, first=1)
        b.step_hosted(X, v, bad)
    # positions only: the velocities and the FIRE scalars stay resident in the handle
    for it in range(4):
        a.step(1)
        b.step_hosted(X, None, None, n_blocks)
        Xa, va = a.get_state()
        assert np.array_equal(X, Xa) and np.array_equal(b.get_state()[1], va), it
    sa, sb = a.get_status(), b.get_status()
    assert (sb.dt, sb.alpha, sb.n_pos, sb.steps, sb.fmax) == (sa.dt, sa.alpha, sa.n_pos, sa.steps, sa.fmax)
    a.close()
    b.close()


def test_hosted_step_and_checkpoint_after_image_control():
    """The state calls on a band whose image count and slot order were changed on the device (cfneb_step_adaptive) and on
    the host (insert / delete): cfneb_step_hosted and a checkpoint resume in a second handle, brought to the same image
    count by the same control calls, stay bit-identical to the resident band."""
    import paper_2510_16721_b200 as cf
    spec, pos, cells = build_workload(1)
    prm = cf.params_for(spec, cell_factor=0.0, max_images=14)
    a = cf.CFNEB(pos, cells, prm)
    b = cf.CFNEB(pos, cells, prm)
    L0 = float(np.sum(a.get_segment_lengths()))
    for g in (a, b):
        g.step_adaptive(6, 3, L0 / 10.0, L0 / 40.0)     # grows the band on the device
        g.insert_image(1)
        g.delete_image(4 if g.get_status().climb_index != 4 else 5)
        g.step(2)
    P = a.P
    assert P == b.P and P > 9
    ck = b.get_checkpoint()
    assert ck["X"].shape[0] == P
    X, v, fire = np.ascontiguousarray(ck["X"]), np.ascontiguousarray(ck["v"]), ck["fire"]
    for it in range(4):
        a.step(1)
        b.step_hosted(X, v, fire, 4)
        Xa, va = a.get_state()
        assert np.array_equal(X, Xa) and np.array_equal(v, va), it
    # resume in a third handle that reached the same P by another route: same endpoints, images inserted anywhere
    c = cf.CFNEB(pos, cells, prm)
    while c.P < P:
        c.insert_image(0)
    ck = a.get_checkpoint()
    c.set_state(ck["X"], ck["v"], ck["X_list"], ck["list_aux"], ck["fire"])
    a.step(5)
    c.step(5)
    assert np.array_equal(a.get_state()[0], c.get_state()[0]) and np.array_equal(a.get_state()[1], c.get_state()[1])
    for g in (a, b, c):
        assert g.get_status().error == 0
        g.close()


@pytest.mark.parametrize("route", ["adaptive", "insert", "reparametrize", "set_state"])
def test_checkpoint_between_calls_carries_the_pending_list_state(route):
    """A checkpoint taken after a call that leaves work for the next cell map -- an image inserted on the device
    (cfneb_step_adaptive ending on its control step) or on the host whose list is still to be built (its X_list row is
    an unused slot's: not a cell), a re-parametrisation or a tracked state import whose displacement the staleness bound
    has not seen yet -- resumes bit for bit in a new handle: list_aux[:, 3] carries that pending state."""
    import paper_2510_16721_b200 as cf
    spec, pos, cells = build_workload(1)
    prm = cf.params_for(spec, cell_factor=0.0, max_images=14)
    a = cf.CFNEB(pos, cells, prm)
    L0 = float(np.sum(a.get_segment_lengths()))
    a.step(4)
    if route == "adaptive":
        a.step_adaptive(6, 3, L0 / 12.0, L0 / 48.0)          # the sixth iteration is followed by an insertion
    elif route == "insert":
        a.insert_image(2)
    elif route == "reparametrize":
        a.reparametrize(True)
    else:
        X, v = a.get_state()
        X[1:-1, :-3] += 1e-3 * np.sin(np.arange(X[1:-1, :-3].size)).reshape(X[1:-1, :-3].shape)
        a.set_state(X, v, None, None, a.get_checkpoint()["fire"])   # lists kept, the move recorded for the next K0
    ck = a.get_checkpoint()
    P = a.P
    pending = ck["list_aux"][:, 3]
    if route in ("adaptive", "insert"):
        assert P > 9 and np.sum(pending < 0) == 1            # the new image: rebuild regardless
    elif route == "reparametrize":
        assert np.any(pending > 0) and np.all(pending >= 0)  # (an image the re-parametrisation left in place carries 0)
    else:
        assert np.all(pending[1:-1] > 0) and np.all(pending >= 0)
    c = cf.CFNEB(pos, cells, prm)
    while c.P < P:
        c.insert_image(0)
    c.step(2)
    c.set_state(ck["X"], ck["v"], ck["X_list"], ck["list_aux"], ck["fire"])
    assert c.get_status().error == 0
    a.step(6)
    c.step(6)
    Xa, va = a.get_state()
    Xc, vc = c.get_state()
    assert np.array_equal(Xa, Xc) and np.array_equal(va, vc)
    sa, sc = a.get_status(), c.get_status()
    assert (sa.dt, sa.alpha, sa.n_pos, sa.fmax, sa.barrier, sa.steps) == (sc.dt, sc.alpha, sc.n_pos, sc.fmax, sc.barrier, sc.steps)
    # and the accounting of the movable images continues identically (the restore itself runs one more cell map of
    # the two endpoints, whose counters play no part in an iteration)
    assert np.array_equal(a.get_checkpoint()["list_aux"][1:-1], c.get_checkpoint()["list_aux"][1:-1])
    a.close()
    c.close()


def test_two_tracked_moves_in_a_row_rebuild_the_lists():
    """Two state imports that keep the lists (cfneb_set_state without X_list), no iteration between them, each inside the
    skin of the state before it but together outside the skin of the build: the second finds the first one's
    displacement still pending and asks for a rebuild instead of keeping the larger of the two."""
    import paper_2510_16721_b200 as cf
    from cfneb_workloads import splitmix64_normals
    from oracle import cfneb as oc
    spec, pos, cells = build_workload(2, 5)
    gpu = cf.CFNEB(pos, cells, cf.params_for(spec, cell_factor=0.0))
    X, _ = gpu.get_state()
    kick = splitmix64_normals(92, X[1:-1, :-3].size).reshape(X[1:-1, :-3].shape)
    kick /= np.max(np.linalg.norm(kick, axis=2))             # largest atomic displacement = 1 (in R~)
    X1 = X.copy()
    X1[1:-1, :-3] += 0.08 * kick
    gpu.set_state(X1)
    aux = gpu.get_checkpoint()["list_aux"]
    assert np.all(aux[1:-1, 3] > 0) and np.all(aux[:, 3] >= 0)   # recorded, no rebuild asked for
    X2 = X1.copy()
    X2[1:-1, :-3] += 0.08 * kick
    gpu.set_state(X2)
    assert np.all(gpu.get_checkpoint()["list_aux"][1:-1, 3] == -1.0)
    r0 = gpu.get_status().rebuilds
    F, V, fneb, E = gpu.get_forces()
    assert gpu.get_status().rebuilds == r0 + 3
    p2, c2, _ = gpu.get_path()
    orc = oc.CFNEB(p2, c2, spec.potential, spec.pot, spec.r_cut, k_spring=spec.k_spring, climb=spec.climb, cell_factor=0.0,
                   fire=spec.fire, skin=spec.skin, max_neighbors=spec.max_neighbors)
    orc.band.forces()
    assert rel(E, orc.band.E) < TOL_FORCE and rel(F[1:-1], orc.evaluator.last["F"]) < TOL_FORCE
    gpu.close()


def test_reparametrize_edge_cases():
    """P = 3 with the single interior image held (nothing moves), P = 3 not held (the image goes to mid arc length),
    the small c0 box with periodic self-images, and two calls in a row (the second is the identity to round-off)."""
    import paper_2510_16721_b200 as cf
    spec, pos, cells = build_workload(0)
    g = cf.CFNEB(pos[[0, 2, 6]], cells[[0, 2, 6]], cf.params_for(spec, cell_factor=0.0, max_images=3))
    g.step(2)
    X0, _ = g.get_state()
    assert g.get_status().climb_index == 1
    g.reparametrize(hold_climbing=True)
    assert np.array_equal(g.get_state()[0], X0)
    g.reparametrize(hold_climbing=False)
    X1, v1 = g.get_state()
    d = g.get_segment_lengths()
    assert abs(d[0] - d[1]) < 0.35 * d.mean() and np.all(v1 == 0)    # on the old polyline at half its arc length
    tot0 = np.linalg.norm(X0[1] - X0[0]) + np.linalg.norm(X0[2] - X0[1])
    assert abs(np.linalg.norm(X1[1] - X0[0]) - 0.5 * tot0) < 1e-9 * tot0 or abs(np.linalg.norm(X1[1] - X0[2]) - 0.5 * tot0) < 1e-9 * tot0
    g.step(2)
    assert g.get_status().error == 0 and np.all(np.isfinite(g.get_path(positions=False)[2]))
    g.close()
    g = cf.CFNEB(pos, cells, cf.params_for(spec, cell_factor=0.0))
    g.step(3)
    g.reparametrize(hold_climbing=False)
    Xa, _ = g.get_state()
    g.reparametrize(hold_climbing=False)
    Xb, _ = g.get_state()
    assert np.max(np.abs(Xb - Xa)) < 1e-3 * np.max(np.abs(Xa)) and np.array_equal(Xb[0], Xa[0]) and np.array_equal(Xb[-1], Xa[-1])
    da = g.get_segment_lengths()
    assert da.max() < 1.05 * da.min()
    g.step(3)
    assert g.get_status().error == 0
    g.close()


def test_history_of_a_long_launch_equals_status_snapshots_step_by_step():
    """cfneb_get_history after ONE cfneb_step(200) -- no host synchronisation in between -- returns, bit for bit, what
    cfneb_get_status reports on a twin band stepped one iteration at a time (fmax, barrier, climbing index, dt, alpha,
    P, rebuild count); the ring keeps the last CFNEB_HISTORY_LEN iterations and refuses what it no longer has."""
    import paper_2510_16721_b200 as cf
    spec, pos, cells = build_workload(0)
    prm = cf.params_for(spec, cell_factor=0.0, rebuild_every=7)
    a, b = cf.CFNEB(pos, cells, prm), cf.CFNEB(pos, cells, prm)
    a.step(200)
    hist = a.get_history(1, 200)
    for s in range(1, 201):
        b.step(1)
        st, e = b.get_status(), hist[s - 1]
        assert (e.step, e.rebuilds, e.n_images, e.climb_index, e.fmax, e.barrier, e.dt, e.alpha) == (
            st.steps, st.rebuilds, st.n_images, st.climb_index, st.fmax, st.barrier, st.dt, st.alpha), s
    assert len({e.dt for e in hist}) > 3 and hist[-1].rebuilds > hist[0].rebuilds and hist[-1].fmax < hist[0].fmax
    tail = a.get_history(150, 51)
    assert [e.step for e in tail] == list(range(150, 201)) and tail[-1].fmax == a.get_status().fmax
    for first, n in ((0, 5), (190, 12), (201, 1)):
        with pytest.raises(cf.CfnebError) as err:
            a.get_history(first, n)
        assert err.value.code == cf.binding.ERANGE
    a.step(cf.HISTORY_LEN)                                   # the ring wraps: iterations 1 .. 200 are gone
    with pytest.raises(cf.CfnebError):
        a.get_history(200, 1)
    wrapped = a.get_history(201, cf.HISTORY_LEN)
    assert [e.step for e in wrapped] == list(range(201, 201 + cf.HISTORY_LEN)) and a.get_status().error == 0
    a.close()
    b.close()


def test_neighbor_list_reuse_equals_fresh_lists():
    """Verlet-list reuse (skin) must not change the result: rebuild_every = 1 forces fresh lists each step."""
    import paper_2510_16721_b200 as cf
    spec, pos, cells = build_workload(2)
    a = cf.CFNEB(pos, cells, cf.params_for(spec, cell_factor=0.0))
    b = cf.CFNEB(pos, cells, cf.params_for(spec, cell_factor=0.0, rebuild_every=1))
    a.step(40)
    b.step(40)
    sa, sb = a.get_status(), b.get_status()
    assert sb.rebuilds > sa.rebuilds
    # list order differs between the two (summation order), so equality is to round-off, not bitwise
    assert rel(a.get_state()[0], b.get_state()[0]) < 1e-11
    a.close()
    b.close()


def test_step_timed_matches_graph_step():
    import paper_2510_16721_b200 as cf
    spec, pos, cells = build_workload(1)
    a = cf.CFNEB(pos, cells, cf.params_for(spec))
    b = cf.CFNEB(pos, cells, cf.params_for(spec))
    a.step(5)
    ms = b.step_timed(5)
    assert ms.shape == (6,) and np.all(ms >= 0) and ms[2] > 0
    assert np.array_equal(a.get_state()[0], b.get_state()[0])
    a.close()
    b.close()


def _triclinic_band(dims, shear, sigma, n_images, seed):
    """A sheared (triclinic) Bain-like band with strongly displaced atoms, some of them outside the cell (unwrapped
    coordinates, A17): bins, periodic shifts and the general formula (taper) paths all see irregular input."""
    from cfneb_workloads import bain_endpoints, linear_path, load_lattice_constants, splitmix64_normals
    lc = load_lattice_constants()
    f0, c0, f1, c1 = bain_endpoints(dims, lc["fs_bcc_a"], lc["fs_fcc_volume_ratio"])
    S = np.eye(3) + np.array(shear, dtype=np.float64)
    c0, c1 = c0 @ S, c1 @ S
    pos, cells = linear_path(f0, c0, f1, c1, n_images, seed, 1e-3)
    kick = splitmix64_normals(seed + 100, pos[0].size).reshape(pos[0].shape) * sigma
    pos = pos + kick[None]                      # the same disorder in every image, endpoints included
    pos[:, ::7] += cells[:, 0:1, :]             # every 7th atom moved out by one lattice vector
    pos[:, 3::11] -= cells[:, 2:3, :] + cells[:, 1:2, :]
    return pos, cells


@pytest.mark.parametrize("dims,n_images", [((3, 3, 4), 5), ((7, 5, 9), 4)])
def test_triclinic_disordered_band_with_unwrapped_atoms(dims, n_images):
    """Edge cases in one band: triclinic cell, N not a multiple of 32 or 128 (72 / 630 atoms), a box narrower than
    2 r_list (explicit periodic shifts, atoms seeing several images of one neighbour) or with >= 3 bins per axis,
    atoms stored outside the cell, disorder of 0.15 A (no two atoms share a shell)."""
    import paper_2510_16721_b200 as cf
    from oracle import cfneb as oc
    from oracle import forcefield as ff
    spec = CONFIGS[2]
    pos, cells = _triclinic_band(dims, [[0, 0.08, -0.05], [0.03, 0, 0.11], [-0.07, 0.02, 0]], 0.15, n_images, 11)
    N = pos.shape[1]
    assert N % 32 != 0
    cap = 256
    orc = oc.CFNEB(pos, cells, spec.potential, spec.pot, spec.r_cut, k_spring=spec.k_spring, climb=True, cell_factor=0.0,
                   fire=spec.fire, skin=spec.skin, max_neighbors=cap)
    gpu = cf.CFNEB(pos, cells, cf.params_for(spec, cell_factor=0.0, max_neighbors=cap, max_images=n_images))
    # neighbour list of an interior image, bit-exact after sorting
    Rt, D = orc.evaluator.deformation(orc.band.X[1])
    cnt, lst, sh = ff.neighbors(Rt, orc.h0, orc.h0 @ D, spec.r_cut + spec.skin, cap)
    gc, gl, gs = gpu.get_neighbors(1)
    assert np.array_equal(gc, cnt)
    assert np.array_equal(sorted_triples(gc, gl, gs), sorted_triples(cnt, lst, sh))
    f_or = orc.band.forces()
    F, V, fneb, E = gpu.get_forces()
    assert rel(E, orc.band.E) < TOL_FORCE
    assert rel(F[1:-1], orc.evaluator.last["F"]) < TOL_FORCE
    assert rel(V[1:-1], orc.evaluator.last["V"]) < TOL_FORCE
    assert rel(fneb[1:-1], np.stack(f_or[1:-1])) < TOL_STEP
    X0, _ = orc.get_state()
    orc.step(3)
    gpu.step(3)
    assert rel(gpu.get_state()[0] - X0, orc.get_state()[0] - X0) < 1e-7
    assert gpu.get_status().error == 0
    gpu.close()


def _unrelaxed_endpoints(kind):
    """Two unrelaxed end states: LJ vacancy hop off the stress-free lattice constant, or a noisy FS Bain pair."""
    from cfneb_workloads import bain_endpoints, splitmix64_normals, vacancy_endpoints_unrelaxed
    if kind == "lj":
        spec = CONFIGS[0]
        f0, cell, f1, _ = vacancy_endpoints_unrelaxed(2, 1.60)
        return spec, f0 @ cell, cell, f1 @ cell, cell.copy()
    spec = CONFIGS[2]
    f0, c0, f1, c1 = bain_endpoints((3, 3, 4), 2.15, 1.05)
    kick = splitmix64_normals(21, f0.size).reshape(f0.shape) * 0.03
    return spec, f0 @ c0 + kick, c0, f1 @ c1 + kick, c1


@pytest.mark.parametrize("kind,mode", [("lj", 1), ("fs", 1), ("lj", 2), ("fs", 2), ("lj", 0)])
def test_relax_endpoints_follows_oracle_trajectory(kind, mode):
    """cfneb_relax_endpoints, 25 updates with no convergence stop: both endpoints follow the oracle's single-structure
    cell-filter FIRE (final endpoint in the frame of the initial cell) step for step, in the Eq. 17 coordinates
    (CELL_B), the Eq. 14 coordinates (CELL_D) and with the cell fixed."""
    import paper_2510_16721_b200 as cf
    from oracle import cfneb as oc
    spec, R0, h0, R1, h1 = _unrelaxed_endpoints(kind)
    n = 25
    kw = dict(fmax_tol=0.0, max_steps=n, cell_factor=0.0, fire=spec.fire, skin=spec.skin, max_neighbors=256, cell_mode=mode)
    Ra, ha, _, _, ita = oc.relax_endpoint(R0, h0, spec.potential, spec.pot, spec.r_cut, **kw)
    Rb, hb, _, _, itb = oc.relax_endpoint(R1, h1, spec.potential, spec.pot, spec.r_cut, h_ref=h0, **kw)
    gpu = cf.CFNEB(np.stack([R0, R1]), np.stack([h0, h1]),
                   cf.params_for(spec, cell_factor=0.0, max_neighbors=256, max_images=5, cell_mode=mode), n_images=5)
    steps, fmax, en = gpu.relax_endpoints(0.0, n, rebuild_band=False)
    assert steps == [n, n]
    pos, cells, E = gpu.get_path()
    assert rel(pos[0] - R0, Ra - R0) < 1e-8 and rel(pos[-1] - R1, Rb - R1) < 1e-8
    if mode == 0:   # cell fixed: nothing but the atoms moves
        assert np.array_equal(ha, h0) and rel(cells[0], h0) < 1e-15 and rel(cells[-1], hb) < 1e-14
    else:
        assert rel(cells[0] - h0, ha - h0) < 1e-8 and rel(cells[-1] - h1, hb - h1) < 1e-8
    assert np.max(np.abs(Ra - R0)) > 1e-3  # something moved
    assert gpu.get_status().error == 0
    gpu.close()


def test_relax_endpoints_converges_and_rebuilds_the_band():
    """To convergence (fmax < 1e-7): energies and update counts of both endpoints equal the oracle's; with
    rebuild_band the band is the one cfneb_create would build from the relaxed endpoints (h0 = relaxed cell of
    image 0, interior linear in X) and then steps with the oracle band built from the exported path."""
    import paper_2510_16721_b200 as cf
    from oracle import cfneb as oc
    spec, R0, h0, R1, h1 = _unrelaxed_endpoints("lj")
    tol = 1e-7
    kw = dict(fmax_tol=tol, max_steps=4000, cell_factor=0.0, fire=spec.fire, skin=spec.skin, max_neighbors=256)
    Ra, ha, Ea, fa, ita = oc.relax_endpoint(R0, h0, spec.potential, spec.pot, spec.r_cut, **kw)
    Rb, hb, Eb, fb, itb = oc.relax_endpoint(R1, h1, spec.potential, spec.pot, spec.r_cut, h_ref=h0, **kw)
    assert fa < tol and fb < tol
    P = 7
    gpu = cf.CFNEB(np.stack([R0, R1]), np.stack([h0, h1]), cf.params_for(spec, cell_factor=0.0, max_neighbors=256, max_images=P),
                   n_images=P)
    steps, fmax, en = gpu.relax_endpoints(tol, 4000, rebuild_band=True)
    assert max(fmax) < tol
    assert abs(steps[0] - ita) <= 1 and abs(steps[1] - itb) <= 1
    assert abs(en[0] - Ea) < 1e-9 * abs(Ea) and abs(en[1] - Eb) < 1e-9 * abs(Eb)
    pos, cells, E = gpu.get_path()
    assert rel(pos[0], Ra) < 1e-7 and rel(cells[0], ha) < 1e-7 and rel(pos[-1], Rb) < 1e-7 and rel(cells[-1], hb) < 1e-7
    X, v = gpu.get_state()
    lam = gpu.get_status().cell_factor
    assert abs(lam - oc.auto_cell_factor(cells[0], R0.shape[0])) < 1e-12 * lam      # lam from the relaxed cell (A13)
    assert np.max(np.abs(X[0][-3:] - lam * np.eye(3))) < 1e-12 * lam                # image 0 is the reference: B = I
    for p in range(1, P - 1):
        t = p / (P - 1)
        assert np.max(np.abs(X[p] - (X[0] + t * (X[-1] - X[0])))) < 1e-12 * np.max(np.abs(X[0]))
    assert np.all(v == 0)
    orc = oc.CFNEB(pos, cells, spec.potential, spec.pot, spec.r_cut, k_spring=spec.k_spring, climb=True, cell_factor=0.0,
                   fire=spec.fire, skin=spec.skin, max_neighbors=256)
    X0, _ = orc.get_state()
    assert rel(X, X0) < 1e-12
    orc.step(4)
    gpu.step(4)
    assert rel(gpu.get_state()[0] - X0, orc.get_state()[0] - X0) < 1e-7
    assert gpu.get_status().error == 0
    gpu.close()


def test_set_path_keeps_lists_inside_the_skin_and_rebuilds_outside():
    """cfneb_set_path adds the distance of the new coordinates from the stored ones to each image's displacement
    bound: a path inside the skin reuses every list, one outside rebuilds; forces match the oracle either way."""
    import paper_2510_16721_b200 as cf
    from cfneb_workloads import splitmix64_normals
    from oracle import cfneb as oc
    spec, pos, cells = build_workload(2, 5)
    prm = cf.params_for(spec, cell_factor=0.0)
    gpu = cf.CFNEB(pos, cells, prm)
    gpu.step(2)
    pos1, cells1, _ = gpu.get_path()

    def oracle_forces(p, c):
        orc = oc.CFNEB(p, c, spec.potential, spec.pot, spec.r_cut, k_spring=spec.k_spring, climb=spec.climb, cell_factor=0.0,
                       fire=spec.fire, skin=spec.skin, max_neighbors=spec.max_neighbors)
        orc.band.forces()
        return orc.band.E, orc.evaluator.last["F"], orc.evaluator.last["V"]

    kick = splitmix64_normals(77, pos1[1:-1].size).reshape(pos1[1:-1].shape)
    for scale, must_rebuild in ((0.01, False), (0.25, True)):  # skin 0.3: 2 x 0.01 x ~3 sigma stays inside, 0.25 does not
        r0 = gpu.get_status().rebuilds
        p2 = pos1.copy()
        p2[1:-1] += scale * kick
        gpu.set_path(p2, cells1)
        F, V, fneb, E = gpu.get_forces()
        rebuilt = gpu.get_status().rebuilds - r0
        assert (rebuilt >= 3) if must_rebuild else (rebuilt == 0), (scale, rebuilt)
        Eo, Fo, Vo = oracle_forces(p2, cells1)
        assert rel(E, Eo) < TOL_FORCE and rel(F[1:-1], Fo) < TOL_FORCE and rel(V[1:-1], Vo) < TOL_FORCE
        assert np.array_equal(gpu.get_path(positions=False)[2], E)  # energies served after the replacement
    assert gpu.get_status().error == 0
    gpu.close()


def test_device_side_adaptive_control_equals_host_side_and_oracle():
    """cfneb_step_adaptive (O9 decided and applied by kernels, no host round trip) against the oracle's
    `step(3); adapt()` loop and against the host-side cfneb_adapt on a second handle: same image counts, same
    coordinates; afterwards host-side insert / delete still work on the refreshed mirrors."""
    import paper_2510_16721_b200 as cf
    spec, orc, gpu = make_pair(1, cell_factor=0.0, max_images=14)
    _, _, host = make_pair(1, cell_factor=0.0, max_images=14)
    orc.max_images = 14
    L0 = float(np.sum(orc.band.segment_lengths()))
    d_insert, d_delete = L0 / 10.0, L0 / 40.0   # the initial spacing L0/8 exceeds d_insert: the band grows
    counts = []
    for cycle in range(4):
        orc.step(3)
        counts.append(orc.adapt(d_insert, d_delete))
        host.step(3)
        assert host.adapt(d_insert, d_delete) == counts[-1]
    gpu.step_adaptive(12, 3, d_insert, d_delete)     # one call, nothing read back in between
    assert sum(c[0] for c in counts) > 0
    assert gpu.P == orc.P == host.P
    Xo, vo = orc.get_state()
    Xg, vg = gpu.get_state()
    Xh, vh = host.get_state()
    assert np.array_equal(Xg, Xh) and np.array_equal(vg, vh)       # device-side == host-side, bit for bit
    assert rel(Xg, Xo) < 1e-11
    # a deletion schedule too: thresholds that prune
    d_insert2, d_delete2 = 10.0 * L0, 2.5 * L0 / (orc.P - 1)
    orc.step(2)
    co = orc.adapt(d_insert2, d_delete2)
    gpu.step_adaptive(2, 2, d_insert2, d_delete2)
    assert co == (0, 1) and gpu.P == orc.P
    assert rel(gpu.get_state()[0], orc.get_state()[0]) < 1e-10
    # host-side control on the refreshed mirrors
    gpu.insert_image(0)
    orc.insert_image(0)
    gpu.step(2)
    orc.step(2)
    assert gpu.P == orc.P and rel(gpu.get_state()[0], orc.get_state()[0]) < 1e-9
    assert gpu.get_status().error == 0
    gpu.close()
    host.close()


def test_c2_converged_bain_barrier_equals_closed_form_saddle():
    """configs[2] (2048 atoms x 16 images) run to fmax < 1e-6 on the device: the barrier is N times the saddle height of
    the closed-form surface E(a, c) (tests/bain_surface.py) -- 252.6056 eV -- to BASELINE.json's 1e-4 eV."""
    import paper_2510_16721_b200 as cf
    from bain_surface import energy_per_atom, saddle
    from cfneb_workloads import load_lattice_constants
    spec, pos, cells = build_workload(2)
    N = pos.shape[1]
    gpu = cf.CFNEB(pos, cells, cf.params_for(spec, cell_factor=0.0))
    for _ in range(40):
        gpu.step(100)
        if gpu.get_status().fmax < 1e-6:
            break
    st = gpu.get_status()
    assert st.error == 0 and st.fmax < 1e-6
    P_, C_, E_ = gpu.get_path()
    a_bcc = load_lattice_constants()["fs_bcc_a"]
    e_bcc = energy_per_atom(a_bcc, a_bcc, spec.pot)
    assert abs(E_[0] / N - e_bcc) < 1e-11
    h = C_[st.climb_index] / np.array(spec.dims, dtype=np.float64)[:, None]
    assert np.abs(h - np.diag(np.diag(h))).max() < 1e-8
    a_s, c_s, e_s, eig = saddle(h[0, 0], h[2, 2], spec.pot)
    assert eig[0] < 0.0 < eig[1]
    assert abs(st.barrier - N * (e_s - e_bcc)) < 1e-4
    assert abs(st.barrier - 252.6056) < 1e-3
    gpu.close()


def test_one_pass_projection_algebra_against_the_materialised_force_to_convergence():
    """K5 never forms f^NEB: it takes f.f and f.v of every image from the ten K4 dot products (f = G + c1 tau+ + c2 tau-).
    That is a difference of terms of the size of G.G, which stays O(10^2) per image on configs[2] while f.f falls with
    fmax^2 -- so its ABSOLUTE error is what is bounded (a few ulp of (|G| + |c1||tau+| + |c2||tau-|)^2),
    and its relative error grows as the band converges.  Compared here, along the whole run to fmax < 1e-6, with the same
    sums over the materialised f^NEB of cfneb_get_forces ("keep a two-pass ... and compare"):
    the absolute bound at every check; 1e-4 relative while fmax > 1e-4 (the convergence criteria of BASELINE.json's
    configs are 1e-3 and 1e-4); and the band totals that drive FIRE stay positive -- K5's clamp of a negative f.f
    does not fire -- and within 20 % down to fmax = 1e-6."""
    import paper_2510_16721_b200 as cf
    spec, pos, cells = build_workload(2)
    gpu = cf.CFNEB(pos, cells, cf.params_for(spec, cell_factor=0.0))
    checks = 0
    for _ in range(40):
        gpu.step(100)
        fmax = gpu.get_status().fmax
        dots, coef, _ = gpu.get_dots(gen_force=False)
        _, _, fneb, _ = gpu.get_forces(forces=False)
        _, v = gpu.get_state()
        d, c1, c2 = dots[1:-1], np.abs(coef[1:-1, 0]), np.abs(coef[1:-1, 1])
        ff_mat = np.sum(fneb[1:-1] ** 2, axis=(1, 2))
        fv_mat = np.sum(fneb[1:-1] * v[1:-1], axis=(1, 2))
        size = np.sqrt(d[:, 5]) + c1 * np.sqrt(d[:, 0]) + c2 * np.sqrt(d[:, 1])      # |G| + |c1| |tau+| + |c2| |tau-|
        assert np.all(np.abs(coef[1:-1, 3] - ff_mat) <= 2e-15 * size ** 2)
        assert np.all(np.abs(coef[1:-1, 2] - fv_mat) <= 2e-15 * size * np.sqrt(d[:, 9]))
        if fmax > 1e-4:
            assert np.max(np.abs(coef[1:-1, 3] - ff_mat) / ff_mat) < 1e-4
        tot1, totm = float(np.sum(coef[1:-1, 3])), float(np.sum(ff_mat))
        assert tot1 > 0.0 and abs(tot1 - totm) < 0.2 * totm, (fmax, tot1, totm)
        checks += 1
        if fmax < 1e-6:
            break
    assert gpu.get_status().fmax < 1e-6 and checks >= 10 and float(np.sum(d[:, 5])) > 1e2   # G.G did not shrink with f
    gpu.close()


@pytest.mark.parametrize("k,over", [(0, dict(skin=0.0)), (2, dict(skin=0.0)), (2, dict(rebuild_every=1)),
                                    (2, dict(max_neighbors=144)), (2, dict(max_neighbors=145)),
                                    (0, dict(max_neighbors=97, skin=0.05))])
def test_list_parameters_at_their_edges(k, over):
    """skin = 0 (r_list = r_cut: no tail buckets, a rebuild whenever anything moves), rebuild_every = 1, and a list
    capacity that is odd or (for the FS band) exactly the largest neighbour count: same forces and steps as the oracle,
    whose own lists use the same skin."""
    import paper_2510_16721_b200 as cf
    from oracle import cfneb as oc
    spec, pos, cells = build_workload(k, 5 if k == 2 else None)
    skin = over.get("skin", spec.skin)
    cap_o = 256
    orc = oc.CFNEB(pos, cells, spec.potential, spec.pot, spec.r_cut, k_spring=spec.k_spring, climb=spec.climb, cell_factor=0.0,
                   fire=spec.fire, skin=skin, max_neighbors=cap_o)
    gpu = cf.CFNEB(pos, cells, cf.params_for(spec, cell_factor=0.0, **over))
    f_or = orc.band.forces()
    F, V, fneb, E = gpu.get_forces()
    assert rel(E, orc.band.E) < TOL_FORCE and rel(F[1:-1], orc.evaluator.last["F"]) < TOL_FORCE
    assert rel(V[1:-1], orc.evaluator.last["V"]) < TOL_FORCE and rel(fneb[1:-1], np.stack(f_or[1:-1])) < TOL_STEP
    X0, _ = orc.get_state()
    orc.step(4)
    gpu.step(4)
    assert rel(gpu.get_state()[0] - X0, orc.get_state()[0] - X0) < 1e-7
    st = gpu.get_status()
    assert st.error == 0
    if "max_neighbors" in over and k == 2:
        assert st.max_neighbors_seen == 144                         # capacity exactly reached (144) or odd, one above (145)
    if over.get("rebuild_every") == 1 or skin == 0.0:
        assert st.rebuilds >= 4 * (pos.shape[0] - 2)
    gpu.close()


def test_list_reuse_under_compression_and_disorder_equals_fresh_lists():
    """The staleness bound at work where it matters: a strongly disordered triclinic band under 80 GPa, whose cells
    shrink by several per cent (pairs come inside r_cut that were outside r_list at the build) while atoms move by
    more than the skin.  Reused lists must give the state that fresh lists (rebuild_every = 1) give, and the reuse
    run must have rebuilt some lists on its own and skipped most."""
    import paper_2510_16721_b200 as cf
    spec = CONFIGS[2]
    pos, cells = _triclinic_band((4, 4, 5), [[0, 0.05, -0.03], [0.02, 0, 0.06], [-0.04, 0.01, 0]], 0.12, 6, 5)
    kw = dict(cell_factor=0.0, max_neighbors=256, max_images=6, pressure=0.5)
    a = cf.CFNEB(pos, cells, cf.params_for(spec, **kw))
    b = cf.CFNEB(pos, cells, cf.params_for(spec, rebuild_every=1, **kw))
    vol0 = abs(np.linalg.det(a.get_path(positions=False)[1][2]))
    n = 120
    a.step(n)
    b.step(n)
    sa, sb = a.get_status(), b.get_status()
    assert sa.error == 0 and sb.error == 0
    movable = pos.shape[0] - 2
    assert sb.rebuilds >= n * movable
    assert 2 * movable < sa.rebuilds < sb.rebuilds // 3          # stale lists were detected, most steps reused theirs
    Xa, Xb = a.get_state()[0], b.get_state()[0]
    X0 = cf.CFNEB(pos, cells, cf.params_for(spec, **kw)).get_state()[0]
    assert np.max(np.abs(Xa[:, :-3] - X0[:, :-3])) > spec.skin    # atoms moved by more than the skin
    vol1 = abs(np.linalg.det(a.get_path(positions=False)[1][2]))
    assert vol1 < 0.97 * vol0                                    # and the cell was compressed
    assert rel(Xa - X0, Xb - X0) < 1e-9
    a.close()
    b.close()


@pytest.mark.parametrize("beta,rho_r0", [(2.7, 2.3), (3.0, 2.1)])
def test_fs_potential_with_general_density_exponent(beta, rho_r0):
    """BASELINE.json's potential has beta = 2 alpha, for which the force kernel shares one exponential between the
    pair and the density term; beta != 2 alpha takes the other template instance (two exponentials), and
    beta = 2 alpha with rho_r0 != r0 exercises the constant factor of the shared form."""
    import paper_2510_16721_b200 as cf
    from cfneb_workloads import fs_params
    from oracle import cfneb as oc
    spec, pos, cells = build_workload(2, 5, dims=(4, 4, 4))
    pot = fs_params(beta=beta, rho_r0=rho_r0)
    orc = oc.CFNEB(pos, cells, spec.potential, pot, spec.r_cut, k_spring=spec.k_spring, climb=True, cell_factor=0.0,
                   fire=spec.fire, skin=spec.skin, max_neighbors=spec.max_neighbors)
    gpu = cf.CFNEB(pos, cells, cf.params_for(spec, cell_factor=0.0, pot=list(pot)))
    f_or = orc.band.forces()
    F, V, fneb, E = gpu.get_forces()
    assert rel(E, orc.band.E) < TOL_FORCE and rel(F[1:-1], orc.evaluator.last["F"]) < TOL_FORCE
    assert rel(V[1:-1], orc.evaluator.last["V"]) < TOL_FORCE and rel(fneb[1:-1], np.stack(f_or[1:-1])) < TOL_STEP
    assert np.max(np.abs(orc.evaluator.last["F"])) > 1e-3     # off the stored lattice constant: real forces
    X0, _ = orc.get_state()
    orc.step(4)
    gpu.step(4)
    assert rel(gpu.get_state()[0] - X0, orc.get_state()[0] - X0) < 1e-7
    assert gpu.get_status().error == 0
    gpu.close()


def test_two_path_replacements_in_a_row_keep_the_lists_valid():
    """Two cfneb_set_path calls with no iteration between them, each inside the skin of the previous path but together
    outside the skin of the coordinates the lists were built at: the staleness bound must see the sum."""
    import paper_2510_16721_b200 as cf
    from cfneb_workloads import splitmix64_normals
    from oracle import cfneb as oc
    spec, pos, cells = build_workload(2, 5)
    gpu = cf.CFNEB(pos, cells, cf.params_for(spec, cell_factor=0.0))
    kick = splitmix64_normals(91, pos[1:-1].size).reshape(pos[1:-1].shape)
    kick /= np.max(np.linalg.norm(kick, axis=2))             # largest atomic displacement = 1
    r0 = gpu.get_status().rebuilds
    p1 = pos.copy()
    p1[1:-1] += 0.10 * kick                                  # 2 x 0.10 < skin 0.3: no rebuild
    gpu.set_path(p1, cells)
    assert gpu.get_status().rebuilds == r0
    p2 = p1.copy()
    p2[1:-1] += 0.10 * kick                                  # again inside the skin of p1, but 2 x 0.20 > 0.3 from the build
    gpu.set_path(p2, cells)
    F, V, fneb, E = gpu.get_forces()
    assert gpu.get_status().rebuilds >= r0 + 3
    orc = oc.CFNEB(p2, cells, spec.potential, spec.pot, spec.r_cut, k_spring=spec.k_spring, climb=spec.climb, cell_factor=0.0,
                   fire=spec.fire, skin=spec.skin, max_neighbors=spec.max_neighbors)
    orc.band.forces()
    assert rel(E, orc.band.E) < TOL_FORCE and rel(F[1:-1], orc.evaluator.last["F"]) < TOL_FORCE
    gpu.close()


def _sw_band(dims, n_images, a=5.35, strain=((0.0, 0.03, 0.0), (0.02, -0.03, 0.0), (0.0, 0.01, 0.04))):
    from cfneb_workloads import diamond_strain_band, sw_params
    pot = sw_params()
    pos, cells = diamond_strain_band(dims, a, n_images, 17, 0.08, strain)
    return pot, pos, cells


@pytest.mark.parametrize("dims,n_images", [((2, 2, 2), 5), ((3, 3, 4), 4)])
def test_stillinger_weber_many_body_forces_and_steps(dims, n_images):
    """The three-body potential through the paper's partial-force formalism (Eq. 5, 8) on the device against the
    oracle: a disordered diamond band under strain; the 64-atom cell is narrower than 3 r_list (explicit periodic
    shifts, mirror entries across the boundary), the 288-atom one uses the binned search."""
    import paper_2510_16721_b200 as cf
    from oracle import cfneb as oc
    pot, pos, cells = _sw_band(dims, n_images)
    rc = pot[2] * pot[1]
    fire = dict(dt0=0.05, dtmax=0.5, maxstep=0.1, nmin=5, finc=1.1, fdec=0.5, astart=0.1, fa=0.99)
    orc = oc.CFNEB(pos, cells, 2, pot, rc, k_spring=1.0, climb=True, cell_factor=0.0, fire=fire, skin=0.3, max_neighbors=64)
    prm = cf.default_params(potential=cf.POT_SW, pot=list(pot), k_spring=1.0, climb=1, cell_factor=0.0, skin=0.3,
                            max_neighbors=64, max_images=n_images, fire=fire)
    gpu = cf.CFNEB(pos, cells, prm)
    f_or = orc.band.forces()
    F, V, fneb, E = gpu.get_forces()
    assert np.max(np.abs(orc.evaluator.last["F"])) > 0.5          # real forces, three-body terms far from zero
    assert rel(E, orc.band.E) < TOL_FORCE
    assert rel(F[1:-1], orc.evaluator.last["F"]) < TOL_FORCE
    assert rel(V[1:-1], orc.evaluator.last["V"]) < TOL_FORCE
    assert rel(fneb[1:-1], np.stack(f_or[1:-1])) < TOL_STEP
    X0 = first_step_exact(orc, gpu)
    orc.step(5)
    gpu.step(5)
    Xo, vo = orc.get_state()
    Xg, vg = gpu.get_state()
    assert rel(Xg - X0, Xo - X0) < 1e-7 and rel(vg, vo) < 1e-7
    st = gpu.get_status()
    assert st.error == 0 and abs(st.barrier - orc.band.barrier) < 1e-9 * max(1.0, abs(orc.band.E[0]))
    gpu.close()


def test_stillinger_weber_step_length_limit_follows_oracle():
    """The step-length limit (A4) on a many-body band: active on every compared iteration (asserted on the oracle)."""
    import paper_2510_16721_b200 as cf
    from oracle import cfneb as oc
    pot, pos, cells = _sw_band((2, 2, 2), 5)
    fire = dict(dt0=0.05, dtmax=0.5, maxstep=1e-5, nmin=5, finc=1.1, fdec=0.5, astart=0.1, fa=0.99)
    orc = record_branches(oc.CFNEB(pos, cells, 2, pot, pot[2] * pot[1], k_spring=1.0, climb=True, cell_factor=0.0, fire=fire,
                                   skin=0.3, max_neighbors=64))
    gpu = cf.CFNEB(pos, cells, cf.default_params(potential=cf.POT_SW, pot=list(pot), k_spring=1.0, climb=1, cell_factor=0.0,
                                                 skin=0.3, max_neighbors=64, max_images=5, fire=fire))
    X0 = first_step_exact(orc, gpu)
    orc.step(4)
    gpu.step(4)
    assert orc.clipped_steps == 5
    Xo, vo = orc.get_state()
    Xg, vg = gpu.get_state()
    assert rel(Xg - X0, Xo - X0) < 1e-7 and rel(vg, vo) < 1e-7
    assert gpu.get_status().error == 0
    gpu.close()


def test_stillinger_weber_band_converges_with_the_oracle():
    """The many-body workload (cfneb_workloads config 5 at 216 atoms x 6 images: relaxed diamond to a generally strained
    cell, no climbing image) run to convergence on the device and by the oracle: same energies along the band,
    equally spaced images, endpoint at the -2 eps per atom of the published parametrisation."""
    import paper_2510_16721_b200 as cf
    from oracle import cfneb as oc
    spec, pos, cells = build_workload(5, 6, dims=(3, 3, 3))
    N = pos.shape[1]
    orc = oc.CFNEB(pos, cells, spec.potential, spec.pot, spec.r_cut, k_spring=spec.k_spring, climb=spec.climb, cell_factor=0.0,
                   fire=spec.fire, skin=spec.skin, max_neighbors=spec.max_neighbors)
    gpu = cf.CFNEB(pos, cells, cf.params_for(spec, cell_factor=0.0, max_images=6))
    orc.step(260)
    gpu.step(260)
    st = gpu.get_status()
    assert st.error == 0 and st.fmax < 1e-6 and orc.band.fmax < 1e-6 and st.climb_index == -1
    Eg = gpu.get_path(positions=False)[2]
    assert np.max(np.abs(Eg - orc.band.E)) < 1e-8
    assert abs(Eg[0] / N + 2.0 * spec.pot[0]) < 2e-4 * spec.pot[0]
    seg = gpu.get_segment_lengths()
    assert np.max(seg) - np.min(seg) < 1e-4 * np.mean(seg)
    gpu.close()


def test_relax_endpoints_stillinger_weber_finds_the_published_diamond():
    """Endpoint relaxation on the device with the many-body potential: diamond compressed to a = 5.30 A (and a noisy,
    stretched copy as the other endpoint) relaxes, cell and atoms together, to the crystal the published constants were
    built for -- -2 eps per atom, a = 5.431 A -- and to the oracle's relaxed energy."""
    import paper_2510_16721_b200 as cf
    from cfneb_workloads import diamond_supercell, splitmix64_normals, sw_params
    from oracle import cfneb as oc
    pot = sw_params()
    rc = pot[2] * pot[1]
    fire = dict(dt0=0.02, dtmax=0.15, maxstep=0.05, nmin=5, finc=1.1, fdec=0.5, astart=0.1, fa=0.99)
    frac, c0 = diamond_supercell(2, 2, 2, 5.30)
    _, c1 = diamond_supercell(2, 2, 2, 5.52)
    N = len(frac)
    R0 = frac @ c0
    R1 = frac @ c1 + 0.03 * splitmix64_normals(3, frac.size).reshape(frac.shape)
    prm = cf.default_params(potential=cf.POT_SW, pot=list(pot), k_spring=1.0, climb=0, cell_factor=0.0, skin=0.3,
                            max_neighbors=64, max_images=4, fire=fire)
    gpu = cf.CFNEB(np.stack([R0, R1]), np.stack([c0, c1]), prm, n_images=4)
    steps, fmax, en = gpu.relax_endpoints(1e-7, 6000, rebuild_band=True)
    assert max(fmax) < 1e-7
    Ra, ha, Ea, fa, ita = oc.relax_endpoint(R0, c0, 2, pot, rc, fmax_tol=1e-7, max_steps=6000, cell_factor=0.0, fire=fire,
                                            skin=0.3, max_neighbors=64)
    assert abs(en[0] - Ea) < 1e-9 * abs(Ea) and abs(steps[0] - ita) <= 1
    pos, cells, E = gpu.get_path()
    for e, h in ((en[0], cells[0]), (en[1], cells[-1])):
        assert abs(e / N + 2.0 * pot[0]) < 2e-4 * pot[0]
        a_eff = abs(np.linalg.det(h)) ** (1.0 / 3.0) / 2.0
        assert abs(a_eff - 5.431) < 2e-3
    assert abs(E[0] - E[-1]) < 1e-6                      # both endpoints are the same crystal: a flat band
    assert gpu.get_status().error == 0
    gpu.close()


@pytest.mark.parametrize("dims,n_images,net", [((2, 2, 2), 5, dict()), ((3, 3, 4), 4, dict()),
                                               ((2, 2, 3), 4, dict(rc=3.6, K=2, M=4, L=2, H=5, seed=7)),
                                               ((2, 2, 2), 3, dict(rc=4.4, K=4, M=1, L=1, H=1, seed=3)),
                                               ((2, 2, 2), 3, dict(rc=5.6, K=3, M=4, L=3, H=8, seed=11))])
def test_descriptor_network_many_body_forces_and_steps(dims, n_images, net):
    """CFNEB_POT_DNN -- the shape of the paper's NEP: radial + angular descriptors into a one-hidden-layer
    network, seeded weights -- through the same partial-force passes (Eq. 5, 8) against the oracle: energies, forces,
    virials, f^NEB, then a few FIRE steps.  Disordered, strained diamond bands with 16 to 46 atoms inside the cut-off;
    the small cells are narrower than 3 r_list (explicit periodic shifts).  Other descriptor counts and network widths
    than the default exercise the index arithmetic."""
    import paper_2510_16721_b200 as cf
    from cfneb_workloads import diamond_strain_band, dn_params
    from oracle import cfneb as oc
    pot = dn_params(**net)
    pos, cells = diamond_strain_band(dims, 5.35, n_images, 23, 0.08, ((0.0, 0.03, 0.0), (0.02, -0.03, 0.0), (0.0, 0.01, 0.04)))
    fire = dict(dt0=0.02, dtmax=0.1, maxstep=0.02, nmin=5, finc=1.1, fdec=0.5, astart=0.1, fa=0.99)
    orc = oc.CFNEB(pos, cells, 3, pot, pot[0], k_spring=1.0, climb=True, cell_factor=0.0, fire=fire, skin=0.3, max_neighbors=96)
    prm = cf.default_params(potential=cf.POT_DNN, pot=list(pot), k_spring=1.0, climb=1, cell_factor=0.0, skin=0.3,
                            max_neighbors=96, max_images=n_images, fire=fire)
    gpu = cf.CFNEB(pos, cells, prm)
    f_or = orc.band.forces()
    F, V, fneb, E = gpu.get_forces()
    assert np.max(np.abs(orc.evaluator.last["F"])) > 1e-3
    assert rel(E, orc.band.E) < TOL_FORCE
    assert rel(F[1:-1], orc.evaluator.last["F"]) < TOL_FORCE
    assert rel(V[1:-1], orc.evaluator.last["V"]) < TOL_FORCE
    assert rel(fneb[1:-1], np.stack(f_or[1:-1])) < TOL_STEP
    X0 = first_step_exact(orc, gpu)
    orc.step(5)
    gpu.step(5)
    Xo, vo = orc.get_state()
    Xg, vg = gpu.get_state()
    assert rel(Xg - X0, Xo - X0) < 1e-7 and rel(vg, vo) < 1e-7
    assert gpu.get_status().error == 0
    gpu.close()


@pytest.mark.parametrize("dims,n_images,net", [
    ((2, 2, 2), 4, dict()),
    ((3, 3, 3), 3, dict()),
    ((2, 2, 3), 3, dict(rc_r=5.2, rc_a=3.2, n_r=3, n_a=2, k_r=5, k_a=4, L=2, H=9, n_types=1, seed=7)),
    ((2, 2, 2), 3, dict(rc_r=4.4, rc_a=4.4, n_r=8, n_a=8, k_r=12, k_a=12, L=4, H=64, n_types=2, seed=3)),
    ((2, 2, 2), 4, dict(rc_r=6.1, rc_a=2.9, n_r=1, n_a=5, k_r=1, k_a=3, L=3, H=2, n_types=2, seed=12))])
def test_nep_shaped_potential_forces_and_steps(dims, n_images, net):
    """CFNEB_POT_NEP -- the shape of the paper's force field proper: two cut-offs, two atom types with type-pair
    expansion coefficients, Legendre orders to 4, tens of neurons per type -- against the oracle: energies, forces,
    virials, f^NEB, one exact step, then five more.  Disordered, strained two-species diamond bands; the default
    shape has 70 atoms inside the radial and 28 inside the angular cut-off; the cells are narrower than 2 r_list
    (atoms see several images of one neighbour).  The other shapes exercise the lane split: one and two passes over
    the angular channels (n_a = 2, 5, 8), the largest network, a single neuron, a single type, rc_a = rc_r."""
    import paper_2510_16721_b200 as cf
    from cfneb_workloads import diamond_strain_band, nep_params, two_sublattice_types
    from oracle import cfneb as oc
    pot = nep_params(**net)
    pos, cells = diamond_strain_band(dims, 5.35, n_images, 29, 0.08, ((0.0, 0.03, 0.0), (0.02, -0.03, 0.0), (0.0, 0.01, 0.04)))
    N = pos.shape[1]
    types = two_sublattice_types(N, int(pot[8]))
    # steps large enough that the displacement (dt0^2 f ~ 1e-5) stands clear of the round-off of the coordinates (~1e-15)
    fire = dict(dt0=0.05, dtmax=0.1, maxstep=0.01, nmin=5, finc=1.1, fdec=0.5, astart=0.1, fa=0.99)
    cap = 320
    orc = oc.CFNEB(pos, cells, 4, pot, pot[0], k_spring=1.0, climb=True, cell_factor=0.0, fire=fire, skin=0.3, max_neighbors=cap,
                   types=types)
    prm = cf.default_params(potential=cf.POT_NEP, pot=list(pot), k_spring=1.0, climb=1, cell_factor=0.0, skin=0.3,
                            max_neighbors=cap, max_images=n_images, fire=fire, types=types)
    gpu = cf.CFNEB(pos, cells, prm)
    f_or = orc.band.forces()
    F, V, fneb, E = gpu.get_forces()
    assert np.max(np.abs(orc.evaluator.last["F"])) > 1e-3
    assert rel(E, orc.band.E) < TOL_FORCE
    assert rel(F[1:-1], orc.evaluator.last["F"]) < TOL_FORCE
    assert rel(V[1:-1], orc.evaluator.last["V"]) < TOL_FORCE
    assert rel(fneb[1:-1], np.stack(f_or[1:-1])) < TOL_STEP
    X0 = first_step_exact(orc, gpu)
    orc.step(5)
    gpu.step(5)
    Xo, vo = orc.get_state()
    Xg, vg = gpu.get_state()
    assert rel(Xg - X0, Xo - X0) < 1e-7 and rel(vg, vo) < 1e-7
    assert gpu.get_status().error == 0
    gpu.close()


def test_nep_shaped_potential_with_the_rest_of_the_path():
    """The NEP-shaped potential through the parts of the path that do not know the potential: external pressure with the
    Eq. 14 cell force, an inserted image, re-parametrisation, endpoint relaxation -- against the oracle."""
    import paper_2510_16721_b200 as cf
    from cfneb_workloads import diamond_strain_band, nep_params, two_sublattice_types
    from oracle import cfneb as oc
    from oracle import cellfilter as ocf
    pot = nep_params(rc_r=5.6, rc_a=3.9, n_r=4, n_a=3, k_r=6, k_a=5, L=4, H=12, n_types=2, seed=5)
    pos, cells = diamond_strain_band((2, 2, 3), 5.35, 5, 31, 0.06, ((0.0, 0.04, 0.0), (0.02, -0.03, 0.0), (0.0, 0.01, 0.05)))
    types = two_sublattice_types(pos.shape[1], 2)
    fire = dict(dt0=0.05, dtmax=0.1, maxstep=0.01, nmin=5, finc=1.1, fdec=0.5, astart=0.1, fa=0.99)
    orc = oc.CFNEB(pos, cells, 4, pot, pot[0], k_spring=1.0, climb=True, cell_factor=0.0, fire=fire, skin=0.3, max_neighbors=256,
                   cell_mode=ocf.CELL_D, pressure=0.05, types=types)
    prm = cf.default_params(potential=cf.POT_NEP, pot=list(pot), k_spring=1.0, climb=1, cell_factor=0.0, skin=0.3,
                            max_neighbors=256, max_images=8, fire=fire, cell_mode=cf.CELL_D, pressure=0.05, types=types)
    gpu = cf.CFNEB(pos, cells, prm)
    f_or = orc.band.forces()
    F, V, fneb, E = gpu.get_forces()
    assert rel(E, orc.band.E) < TOL_FORCE and rel(V[1:-1], orc.evaluator.last["V"]) < TOL_FORCE
    assert rel(fneb[1:-1], np.stack(f_or[1:-1])) < TOL_STEP
    X0 = first_step_exact(orc, gpu)
    orc.step(3)
    gpu.step(3)
    assert rel(gpu.get_state()[0] - X0, orc.get_state()[0] - X0) < 1e-7
    p = int(np.argmax(gpu.get_segment_lengths()))
    gpu.insert_image(p)
    orc.insert_image(p)
    orc.step(2)
    gpu.step(2)
    orc.reparametrize(hold_climbing=True)
    gpu.reparametrize(hold_climbing=True)
    orc.step(2)
    gpu.step(2)
    Xo, Xg = orc.get_state()[0], gpu.get_state()[0]
    assert Xg.shape == Xo.shape and rel(Xg, Xo) < 1e-9
    assert gpu.get_status().error == 0
    gpu.close()
    kw = dict(fmax_tol=0.0, max_steps=10, cell_factor=0.0, fire=fire, skin=0.3, max_neighbors=256, types=types)
    Ra, ha, _, _, _ = oc.relax_endpoint(pos[0], cells[0], 4, pot, pot[0], **kw)
    prm2 = cf.default_params(potential=cf.POT_NEP, pot=list(pot), k_spring=1.0, climb=0, cell_factor=0.0, skin=0.3,
                             max_neighbors=256, max_images=4, fire=fire, types=types)
    gpu = cf.CFNEB(np.stack([pos[0], pos[-1]]), np.stack([cells[0], cells[-1]]), prm2, n_images=4)
    steps, fmax, en = gpu.relax_endpoints(0.0, 10, rebuild_band=False)
    p2, c2, _ = gpu.get_path()
    assert steps == [10, 10]
    assert rel(p2[0] - pos[0], Ra - pos[0]) < 1e-8 and rel(c2[0] - cells[0], ha - cells[0]) < 1e-8
    assert gpu.get_status().error == 0
    gpu.close()


def test_nep_shaped_potential_hosted_step_and_resume():
    """The four kernels of the NEP-shaped potential under the image-block selector of cfneb_step_hosted (each uploaded
    block evaluated on its own) and under the list replay of cfneb_set_state: bit-identical to the resident band."""
    import paper_2510_16721_b200 as cf
    from cfneb_workloads import diamond_strain_band, nep_params, two_sublattice_types
    pot = nep_params(rc_r=5.6, rc_a=3.9, n_r=4, n_a=3, k_r=6, k_a=5, L=4, H=12, n_types=2, seed=5)
    pos, cells = diamond_strain_band((2, 2, 3), 5.35, 7, 33, 0.06, ((0.0, 0.04, 0.0), (0.02, -0.03, 0.0), (0.0, 0.01, 0.05)))
    types = two_sublattice_types(pos.shape[1], 2)
    fire = dict(dt0=0.05, dtmax=0.1, maxstep=0.01, nmin=5, finc=1.1, fdec=0.5, astart=0.1, fa=0.99)
    prm = cf.default_params(potential=cf.POT_NEP, pot=list(pot), k_spring=1.0, climb=1, cell_factor=0.0, skin=0.3,
                            max_neighbors=256, max_images=7, fire=fire, types=types)
    a, b = cf.CFNEB(pos, cells, prm), cf.CFNEB(pos, cells, prm)
    a.step(3)
    b.step(3)
    ck = b.get_checkpoint()
    X, v, fs = np.ascontiguousarray(ck["X"]), np.ascontiguousarray(ck["v"]), ck["fire"]
    for it in range(3):
        a.step(1)
        b.step_hosted(X, v, fs, 3)  # 5 movable images in blocks of 2, 2, 1
        Xa, va = a.get_state()
        assert np.array_equal(X, Xa) and np.array_equal(v, va), it
    ck = a.get_checkpoint()
    c = cf.CFNEB(pos, cells, prm)
    c.set_state(ck["X"], ck["v"], ck["X_list"], ck["list_aux"], ck["fire"])
    a.step(4)
    c.step(4)
    assert np.array_equal(a.get_state()[0], c.get_state()[0]) and np.array_equal(a.get_state()[1], c.get_state()[1])
    for g in (a, b, c):
        assert g.get_status().error == 0
        g.close()


def test_nep_shaped_potential_parameter_errors():
    """Out-of-range shapes are refused (workspace size 0); a type outside [0, n_types) is refused by cfneb_create."""
    import paper_2510_16721_b200 as cf
    from cfneb_workloads import diamond_strain_band, nep_params
    for bad in (dict(L=5), dict(n_r=9), dict(n_a=0), dict(k_r=13), dict(H=65), dict(n_types=3), dict(rc_a=8.0), dict(rc_r=0.0)):
        prm = cf.default_params(potential=cf.POT_NEP, pot=list(nep_params(**bad)), max_images=3)
        assert cf.binding.workspace_bytes(64, prm) == 0
    pos, cells = diamond_strain_band((2, 2, 2), 5.35, 3, 1, 0.05, ((0.0, 0.02, 0.0), (0.0, 0.0, 0.0), (0.0, 0.0, 0.02)))
    types = np.zeros(pos.shape[1], dtype=np.int32)
    types[5] = 2
    prm = cf.default_params(potential=cf.POT_NEP, pot=list(nep_params()), max_images=3, max_neighbors=320, types=types)
    with pytest.raises(cf.CfnebError) as e:
        cf.CFNEB(pos, cells, prm)
    assert e.value.code == cf.binding.EINVAL


def test_descriptor_network_parameter_errors():
    """Out-of-range network shapes are refused (workspace size 0)."""
    import paper_2510_16721_b200 as cf
    from cfneb_workloads import dn_params
    for bad in (dict(K=5), dict(M=0), dict(L=4), dict(H=9), dict(K=0), dict(rc=0.0)):
        pot = dn_params(**bad)
        prm = cf.default_params(potential=cf.POT_DNN, pot=list(pot), max_images=3)
        assert cf.binding.workspace_bytes(64, prm) == 0


def test_descriptor_network_with_the_rest_of_the_path():
    """The descriptor-network potential through the parts of the path that do not know the potential: external
    pressure with the Eq. 14 cell force (CELL_D), device-side adaptive control, and the endpoint relaxation -- each
    against the oracle on a disordered strained diamond band."""
    import paper_2510_16721_b200 as cf
    from cfneb_workloads import diamond_strain_band, dn_params
    from oracle import cfneb as oc
    from oracle import cellfilter as ocf
    pot = dn_params(rc=3.9, K=3, M=2, L=3, H=6, seed=5)
    pos, cells = diamond_strain_band((2, 2, 3), 5.35, 5, 31, 0.06, ((0.0, 0.04, 0.0), (0.02, -0.03, 0.0), (0.0, 0.01, 0.05)))
    fire = dict(dt0=0.02, dtmax=0.1, maxstep=0.02, nmin=5, finc=1.1, fdec=0.5, astart=0.1, fa=0.99)
    # pressure + CELL_D
    orc = oc.CFNEB(pos, cells, 3, pot, pot[0], k_spring=1.0, climb=True, cell_factor=0.0, fire=fire, skin=0.3, max_neighbors=96,
                   cell_mode=ocf.CELL_D, pressure=0.05)
    prm = cf.default_params(potential=cf.POT_DNN, pot=list(pot), k_spring=1.0, climb=1, cell_factor=0.0, skin=0.3,
                            max_neighbors=96, max_images=8, fire=fire, cell_mode=cf.CELL_D, pressure=0.05)
    gpu = cf.CFNEB(pos, cells, prm)
    f_or = orc.band.forces()
    F, V, fneb, E = gpu.get_forces()
    assert rel(E, orc.band.E) < TOL_FORCE and rel(V[1:-1], orc.evaluator.last["V"]) < TOL_FORCE
    assert rel(fneb[1:-1], np.stack(f_or[1:-1])) < TOL_STEP
    X0 = first_step_exact(orc, gpu)
    orc.step(4)
    gpu.step(4)
    assert rel(gpu.get_state()[0] - X0, orc.get_state()[0] - X0) < 1e-7
    # an inserted image is evaluated with the same kernels
    seg = gpu.get_segment_lengths()
    p = int(np.argmax(seg))
    gpu.insert_image(p)
    orc.insert_image(p)
    orc.step(3)
    gpu.step(3)
    Xo, Xg = orc.get_state()[0], gpu.get_state()[0]
    assert Xg.shape == Xo.shape and rel(Xg, Xo) < 1e-9
    assert gpu.get_status().error == 0
    gpu.close()
    # endpoint relaxation, 15 updates
    kw = dict(fmax_tol=0.0, max_steps=15, cell_factor=0.0, fire=fire, skin=0.3, max_neighbors=96)
    Ra, ha, _, _, _ = oc.relax_endpoint(pos[0], cells[0], 3, pot, pot[0], **kw)
    prm2 = cf.default_params(potential=cf.POT_DNN, pot=list(pot), k_spring=1.0, climb=0, cell_factor=0.0, skin=0.3,
                             max_neighbors=96, max_images=4, fire=fire)
    gpu = cf.CFNEB(np.stack([pos[0], pos[-1]]), np.stack([cells[0], cells[-1]]), prm2, n_images=4)
    steps, fmax, en = gpu.relax_endpoints(0.0, 15, rebuild_band=False)
    p2, c2, _ = gpu.get_path()
    assert steps == [15, 15]
    assert rel(p2[0] - pos[0], Ra - pos[0]) < 1e-8 and rel(c2[0] - cells[0], ha - cells[0]) < 1e-8
    assert gpu.get_status().error == 0
    gpu.close()
