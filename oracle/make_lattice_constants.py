"""Write cfneb_workloads/lattice_constants.json -- calls only oracle/ (and the lattice builders).

BASELINE.json configs: "Lattice constant set by oracle 1-D minimisation of cohesive energy" (configs[0]);
"Both endpoints cell-relaxed" (configs[2-4]).  For perfect Bravais lattices the forces vanish by symmetry
and the stress is isotropic by cubic symmetry, so the cell-relaxed endpoint is the lattice constant with
tr V = 0 (dE/da = 0, Eq. 3): found by bisection on tr V(a) of the oracle.

Run:  python -m oracle.make_lattice_constants
"""
import json
import os

import numpy as np

from cfneb_workloads import bain_final_cell, bcc_supercell, fcc_supercell, fs_params, lj_params
from oracle import forcefield as ff


def trace_virial(frac, cell, kind, pot, rc):
    nb = ff.neighbors(frac @ cell, cell, cell, rc, 512, brute=False)
    E, F, V = ff.energy_force_virial(frac @ cell, cell, cell, kind, pot, nb)
    return np.trace(V), E / len(frac), np.abs(F).max(), int(nb[0][0])


def bisect(fn, lo, hi):
    flo = fn(lo)
    assert flo * fn(hi) < 0
    for _ in range(200):
        mid = 0.5 * (lo + hi)
        if mid == lo or mid == hi:
            break
        fm = fn(mid)
        if (fm > 0) == (flo > 0):
            lo, flo = mid, fm
        else:
            hi = mid
    return 0.5 * (lo + hi)


def main():
    out = {}
    lj = lambda a: trace_virial(*fcc_supercell(2, 2, 2, a), 0, lj_params(), 2.5)
    a = bisect(lambda x: lj(x)[0], 1.45, 1.70)
    out["lj_fcc_a"] = a
    out["lj_fcc_e_coh"] = lj(a)[1]
    out["lj_fcc_neighbors"] = lj(a)[3]

    fs = lambda a: trace_virial(*bcc_supercell(3, 3, 3, a), 1, fs_params(), 5.0)
    a = bisect(lambda x: fs(x)[0], 1.9, 2.5)
    out["fs_bcc_a"] = a
    out["fs_bcc_e_coh"] = fs(a)[1]
    out["fs_bcc_neighbors"] = fs(a)[3]

    def fs_fcc(ratio):
        frac, cell = bcc_supercell(3, 3, 3, out["fs_bcc_a"])
        return trace_virial(frac, bain_final_cell(cell, ratio), 1, fs_params(), 5.0)

    r = bisect(lambda x: fs_fcc(x)[0], 0.9, 1.3)
    out["fs_fcc_volume_ratio"] = r
    out["fs_fcc_e_coh"] = fs_fcc(r)[1]
    out["fs_fcc_neighbors"] = fs_fcc(r)[3]
    out["_written_by"] = "python -m oracle.make_lattice_constants (bisection on tr V = 0 of the oracle)"
    path = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "cfneb_workloads",
                        "lattice_constants.json")
    with open(path, "w") as fh:
        json.dump(out, fh, indent=1)
    print(json.dumps(out, indent=1))


if __name__ == "__main__":
    main()
