"""Writes the stored expected values under tests/golden/ by calling ONLY oracle/ (tier-1 brute-force full CI) on the
seeded generators of synth/.  Nothing here imports the CUDA package.  Run: python tests/golden/make_golden.py

config1_fci.txt - BASELINE.json configs[0] (PPP naphthalene CAS(10,10), 2Sz = 0, FCI dimension 63504, readings S6-S9
of DESIGN.md): E_core, E_el(FCI), E_total, Tr gamma and the natural occupations of the FCI 1-RDM (Eq. 9).
The total energy is seed independent (invariant under the exp(kappa) rotation) and agrees with the survey's
independent probe value -0.8822829988 Eh."""
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))
from oracle import fci  # noqa: E402
from synth import make_config  # noqa: E402


def main():
    cfg = make_config(1)
    sp = fci.FCISpace(cfg["k"], cfg["n_elec"], 0)
    e, c = sp.ground_state(cfg["h"], cfg["eri"], tol=1e-12)
    g, G = sp.rdm12(c)
    occ = np.sort(np.linalg.eigvalsh(g))[::-1]
    with open(os.path.join(HERE, "config1_fci.txt"), "w") as f:
        f.write("# written by tests/golden/make_golden.py from oracle/fci.py (brute-force FCI, dim %d)\n" % sp.dim)
        f.write("e_core %.10f\n" % cfg["e_core"])
        f.write("e_el_fci %.10f\n" % e)
        f.write("e_total_fci %.10f\n" % (e + cfg["e_core"]))
        f.write("trace_gamma %.10f\n" % np.trace(g))
        f.write("natural_occupations " + " ".join("%.8f" % x for x in occ) + "\n")


if __name__ == "__main__":
    main()
