"""Write cfneb_workloads/vacancy_endpoints_c{0,1}.json -- calls only oracle/ (and the lattice builders).

BASELINE.json configs[0-1]: "Both endpoints are relaxed by cell-filter FIRE to max force 1e-4."  The
relaxation is the oracle's relax_endpoint (O0-O4 + O7 with f = G); it is run to 1e-7 so that the stored
endpoints satisfy the config's 1e-4 with margin.  Stored values: Cartesian positions and cell of both endpoints,
their energies and the residual max generalized force.  Inputs to BOTH the oracle and the CUDA path.

Run:  python -m oracle.make_relaxed_endpoints
"""
import json
import os

import numpy as np

from cfneb_workloads import CONFIGS, load_lattice_constants, vacancy_endpoints_unrelaxed
from oracle import cfneb as oc


def main():
    a = load_lattice_constants()["lj_fcc_a"]
    root = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "cfneb_workloads")
    for k in (0, 1):
        spec = CONFIGS[k]
        n = spec.dims[0]
        fi, cell, ffin, _ = vacancy_endpoints_unrelaxed(n, a)
        out = {"_written_by": "python -m oracle.make_relaxed_endpoints (oracle cell-filter FIRE, fmax < 1e-7)",
               "config": spec.name, "lattice_constant": a}
        for tag, frac in (("init", fi), ("final", ffin)):
            R, h, E, fm, it = oc.relax_endpoint(frac @ cell, cell, spec.potential, spec.pot, spec.r_cut, fmax_tol=1e-7,
                                                max_steps=50000, fire=spec.fire)
            assert fm < 1e-7, (spec.name, tag, fm)
            out["pos_" + tag] = [[float(repr(x)) for x in row] for row in R.tolist()]
            out["cell_" + tag] = h.tolist()
            out["energy_" + tag] = E
            out["fmax_" + tag] = fm
            print(spec.name, tag, "E =", E, "fmax =", fm, "steps =", it)
        with open(os.path.join(root, "vacancy_endpoints_c%d.json" % k), "w") as fh:
            json.dump(out, fh)


if __name__ == "__main__":
    main()
