"""CPU oracle for the CFNEB hot path -- TEST INFRASTRUCTURE ONLY.

A plain, slow, fp64 restatement of what arXiv:2510.16721 (CFNEB) defines, written from
the paper (/root/reference/PAPER.md, cited as P:line) and from the readings in
SURVEY.md §8(c) / DESIGN.md.  It shares no code with the CUDA path
(`paper_2510_16721_b200/`) and neither imports the other; only `cfneb_workloads`
(seeded input generators, no method arithmetic) serves both.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` / `--impl reference`
legs may import, call, link or execute anything under `oracle/`.

Modules
  forcefield.c / forcefield.py   O2 neighbours (brute force = definition; cell list), O3 potentials (LJ shifted
                                 force, Finnis-Sinclair type, Stillinger-Weber, descriptor network of NEP's
                                 shape with seeded weights), forces, virial (Eq. 4-9)
  cellfilter.py                  O0 input mapping, O1 cell map D = sqrt(B), O4 generalized force (Eq. 10-17)
  neb.py                         O5 improved tangent, O6 NEB / climbing-image force (Eq. 1), O7 FIRE,
                                 O8 measures; generic over a band of n-dof points with a callback
  cfneb.py                       the crystal band: O0-O9 put together, one `step()` = one CFNEB iteration
  mullerbrown.py                 analytic 2-D Mueller-Brown surface (pin for neb.py)

Parity pins: see DESIGN.md section 4.  The Bain-path bands (c2-c4) are pinned by the saddle of the closed-form
lattice-sum surface E(a, c) (tests/bain_surface.py).  The adaptive insertion/deletion rule (O9) is a reading of
P:128 (the paper states the principle only); it is pinned by a hand-worked band whose expected deletion, insertion
and order are written out from the rule's text (tests/test_oracle_cfneb.py).  No function here is unpinned.
"""
