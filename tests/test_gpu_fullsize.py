"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times (configs[3], configs[4]; the
many-body workloads 5 and 6 at their full atom count).

configs[4] (101 306 atoms x 100 images): the oracle is run on ALL images with every host core (one evaluation of
the band at construction + one full step: about a minute on 16 cores), and every output is compared element by
element: energies, per-atom forces, virials, f^NEB, then X and v after one full iteration (K0-K6), then the
neighbour list of one mid-path image, bit-exact after sorting.

configs[3] (9 826 atoms, 12 -> up to 32 images, adaptive): the GPU band and the oracle band run the same schedule
(10 steps, adapt, ...) with the DESIGN.md thresholds; the image count, the inserted / deleted positions and the
coordinates must agree after every control step.
"""
import os

import numpy as np
import pytest

from cfneb_workloads import build_workload

pytestmark = pytest.mark.gpu

TOL_FORCE = 1e-10
TOL_STEP = 1e-9


def rel(a, b):
    a, b = np.asarray(a), np.asarray(b)
    s = np.max(np.abs(b))
    return float(np.max(np.abs(a - b)) / (s if s > 0 else 1.0))


def host_threads():
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


def test_c4_full_size_forces_and_one_step():
    import paper_2510_16721_b200 as cf
    from oracle import cfneb as oc
    from oracle import forcefield as ff
    spec, pos, cells = build_workload(4)
    P, N = pos.shape[0], pos.shape[1]
    assert (N, P) == (101306, 100)
    orc = oc.CFNEB(pos, cells, spec.potential, spec.pot, spec.r_cut, k_spring=spec.k_spring, climb=spec.climb,
                   cell_factor=0.0, fire=spec.fire, skin=spec.skin, max_neighbors=spec.max_neighbors,
                   threads=host_threads())
    gpu = cf.CFNEB(pos, cells, cf.params_for(spec, cell_factor=0.0))  # the band bench.py builds
    f_or = orc.band.forces()
    last = orc.evaluator.last
    F, V, fneb, E = gpu.get_forces()
    assert rel(E, orc.band.E) < TOL_FORCE
    assert rel(V[1:-1], last["V"]) < TOL_FORCE
    worst_f = max(rel(F[p], last["F"][p - 1]) for p in range(1, P - 1))
    assert worst_f < TOL_FORCE, worst_f
    # f^NEB of EVERY image against the untouched oracle band at 1e-9.  At an energy extremum the improved tangent (O5)
    # mixes tau+ and tau- with the weights |E_{p+-1} - E_p|: differences of ~0.3 eV between totals of ~9e5 eV, so the
    # energies must agree to about one ulp (1.2e-10 eV) for the weights to agree to 1e-9.  Both sides carry the
    # total in extended precision (the oracle in long double, the kernels in two doubles: block_sum_dd), so each
    # is the correctly rounded sum of its own site energies; measured: <= 1 ulp on the interior images, 3 ulp on the
    # perfect-lattice endpoint (identical site energies, identical per-atom rounding), f^NEB 5e-11 at the extremum.
    Eo = orc.band.E
    assert np.max(np.abs(E - Eo)) < 8 * np.spacing(np.max(np.abs(Eo)))
    n_mixed = 0
    for p in range(1, P - 1):
        upwind = (Eo[p + 1] > Eo[p] > Eo[p - 1]) or (Eo[p + 1] < Eo[p] < Eo[p - 1])
        n_mixed += 0 if upwind else 1
        assert rel(fneb[p], f_or[p]) < TOL_STEP, (p, upwind)
    assert 1 <= n_mixed <= 3  # the Bain band has one maximum (the climbing image): the energy-weighted branch is exercised
    st = gpu.get_status()
    assert st.climb_index == orc.band.pstar
    # the energies that decide tangent branches and the climbing image are not within round-off of a tie (A24)
    dE = np.abs(np.diff(orc.band.E))
    assert dE.min() > 1e-8 * np.abs(orc.band.E).max()
    del F, V, fneb, f_or

    # neighbour list of one mid-path image, bit-exact after sorting (counts and (j, shift) sets per atom)
    image = P // 2
    Rt, D = orc.evaluator.deformation(orc.band.X[image])
    cnt, lst, sh = ff.neighbors(Rt, orc.h0, orc.h0 @ D, spec.r_cut + spec.skin, spec.max_neighbors)
    gc, gl, gs = gpu.get_neighbors(image)
    assert np.array_equal(gc, cnt)
    key_o = np.where(lst >= 0, lst.astype(np.int64) * 512 + (sh[..., 0] + 4) * 64 + (sh[..., 1] + 4) * 8 + (sh[..., 2] + 4), -1)
    key_g = np.where(gl >= 0, gl.astype(np.int64) * 512 + (gs[..., 0] + 4) * 64 + (gs[..., 1] + 4) * 8 + (gs[..., 2] + 4), -1)
    assert np.array_equal(np.sort(key_g, axis=1), np.sort(key_o, axis=1))
    del key_o, key_g, lst, sh, gl, gs

    # one full iteration
    X0, _ = orc.get_state()
    orc.step(1)
    gpu.step(1)
    Xo, vo = orc.get_state()
    Xg, vg = gpu.get_state()
    assert rel(Xg - X0, Xo - X0) < TOL_STEP
    assert rel(vg, vo) < TOL_STEP
    st = gpu.get_status()
    assert st.error == 0 and st.steps == 1
    assert abs(st.fmax - orc.band.fmax) <= 1e-8 * orc.band.fmax
    gpu.close()


def test_c3_adaptive_band_follows_oracle():
    import paper_2510_16721_b200 as cf
    from oracle import cfneb as oc
    spec, pos, cells = build_workload(3)
    P0, N = pos.shape[0], pos.shape[1]
    assert (N, P0) == (9826, 12)
    max_images = 32
    orc = oc.CFNEB(pos, cells, spec.potential, spec.pot, spec.r_cut, k_spring=spec.k_spring, climb=spec.climb,
                   cell_factor=0.0, fire=spec.fire, skin=spec.skin, max_neighbors=spec.max_neighbors,
                   threads=host_threads())
    orc.max_images = max_images
    gpu = cf.CFNEB(pos, cells, cf.params_for(spec, cell_factor=0.0, max_images=max_images))
    L0 = float(np.sum(orc.band.segment_lengths()))
    assert abs(float(np.sum(gpu.get_segment_lengths())) - L0) < 1e-10 * L0
    d_insert, d_delete = L0 / 28.0, L0 / 120.0  # DESIGN.md section 7 (reading A16)
    grew = 0
    for cycle in range(4):
        orc.step(3)
        gpu.step(3)
        assert rel(gpu.get_segment_lengths(), orc.band.segment_lengths()) < 1e-9
        ro, rg = orc.adapt(d_insert, d_delete), gpu.adapt(d_insert, d_delete)
        assert ro == rg, (cycle, ro, rg)
        grew += rg[0] - rg[1]
        assert gpu.P == orc.P == P0 + grew
        Xo, vo = orc.get_state()
        Xg, vg = gpu.get_state()
        assert rel(Xg, Xo) < 1e-11
        if rg != (0, 0):
            assert np.all(vg == 0)
    assert grew > 0  # the initial spacing L0/11 exceeds d_insert = L0/28: the band must grow
    orc.step(2)
    gpu.step(2)
    assert rel(gpu.get_state()[0], orc.get_state()[0]) < 1e-10
    assert gpu.get_status().error == 0
    gpu.close()


def test_c4_long_run_survives_equal_energy_images():
    """A 100-image band of a perfect crystal parks several images at the bottom of the end basins; after ~960
    iterations three consecutive energies agree to the last bit and the weights of the improved tangent vanish
    (reading A26: bisector).  The run must go on: 1100 iterations, no device error, finite state, BJ.configs[4]'s
    500-step throughput run well inside."""
    import paper_2510_16721_b200 as cf
    spec, pos, cells = build_workload(4)
    gpu = cf.CFNEB(pos, cells, cf.params_for(spec, cell_factor=0.0))
    gpu.step(1100)
    st = gpu.get_status()
    assert st.error == 0 and st.steps == 1100
    assert np.isfinite(st.fmax) and np.isfinite(st.barrier)
    E = gpu.get_path(positions=False)[2]
    assert np.all(np.isfinite(E))
    seg = gpu.get_segment_lengths()
    assert seg.min() > 0.0
    gpu.close()


@pytest.mark.parametrize("k", [5, 6, 8])
def test_many_body_workloads_at_full_atom_count(k):
    """The many-body workloads bench.py --config 5 / 6 / 8 times (32 768 atoms; Stillinger-Weber, the descriptor
    network, and the NEP-shaped potential with two cut-offs and two atom types) at their full atom count in the same launch configuration, on the first, two mid-path and
    the last image of the 32: energies, per-atom forces, virials and f^NEB element by element, then two full steps."""
    import paper_2510_16721_b200 as cf
    from oracle import cfneb as oc
    spec, pos, cells = build_workload(k)
    idx = [0, 15, 16, spec.n_images - 1]
    pos, cells = pos[idx], cells[idx]
    orc = oc.CFNEB(pos, cells, spec.potential, spec.pot, spec.r_cut, k_spring=spec.k_spring, climb=spec.climb, cell_factor=0.0,
                   fire=spec.fire, skin=spec.skin, max_neighbors=spec.max_neighbors, threads=min(4, host_threads()),
                   types=spec.types)
    gpu = cf.CFNEB(pos, cells, cf.params_for(spec, cell_factor=0.0, max_images=4))
    f_or = orc.band.forces()
    F, V, fneb, E = gpu.get_forces()
    assert rel(E, orc.band.E) < TOL_FORCE
    assert rel(F[1:-1], orc.evaluator.last["F"]) < TOL_FORCE
    assert rel(V[1:-1], orc.evaluator.last["V"]) < TOL_FORCE
    assert rel(fneb[1:-1], np.stack(f_or[1:-1])) < TOL_STEP
    X0, _ = orc.get_state()
    orc.step(2)
    gpu.step(2)
    Xo, vo = orc.get_state()
    Xg, vg = gpu.get_state()
    assert rel(Xg - X0, Xo - X0) < 1e-8 and rel(vg, vo) < 1e-8
    assert gpu.get_status().error == 0
    gpu.close()
