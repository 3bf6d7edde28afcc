"""Writes the stored expected values under tests/golden/ -- calls ONLY oracle/ (and the seeded
input generators in workloads/, which hold no method arithmetic).  Re-run after a justified change
of the oracle:  python tests/golden/make_golden.py

PAPER.md prints no value for any structure, so these fixtures are regression
pins of the oracle itself (its correctness is pinned by tests/test_oracle_pins.py) and fixed
reference points for the CUDA parity tests.  Definitions: BASELINE.json north_star; readings in
DESIGN.md section 2.
"""
import json
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

from oracle import basis, mtp            # noqa: E402
from workloads import random_cluster     # noqa: E402


def cluster_case(lev, n_mu, seed, n_atoms, n_species):
    pos, types, box = random_cluster(seed, n_atoms, 11.0, n_species=n_species)
    off, idx, shift = mtp.brute_force_neighbours(pos, box, 5.0)
    rng = np.random.default_rng(seed + 1)
    nb = len(basis.basis_functions(lev))
    c = rng.uniform(-0.1, 0.1, (n_species, n_species, n_mu, 8))
    xi0 = rng.uniform(-0.1, 0.1, n_species)
    xi = rng.uniform(-0.1, 0.1, nb)
    pot = mtp.Potential(lev, n_mu, 8, 2.0, 5.0, c, xi0, xi)
    out = mtp.evaluate(pot, pos, types, box, off, idx, shift)
    return dict(lev=lev, n_mu=n_mu, seed=seed, n_atoms=int(pos.shape[0]), n_species=n_species,
                nnz=int(idx.shape[0]), E=float(out["E"]), E_i=out["E_i"].tolist(), F=out["F"].tolist(),
                virial=mtp.virial6(out["W"]).tolist(), B_atom0=out["B"][0].tolist())


def main():
    cases = [cluster_case(10, 3, 101, 12, 2), cluster_case(16, 4, 102, 9, 1)]
    with open(os.path.join(HERE, "cluster_cases.json"), "w") as f:
        json.dump(dict(source="tests/golden/make_golden.py (oracle/ only); north_star definitions, DESIGN.md readings G1-G24",
                       cases=cases), f, indent=1)
    counts = {str(lev): len(basis.basis_functions(lev)) for lev in range(2, 26, 2)}
    with open(os.path.join(HERE, "basis_counts.txt"), "w") as f:
        f.write("# lev_max n_basis -- level rule lev(M_{mu,nu}) = 2 + 4 mu + nu, BASELINE.json north_star; reading G9\n")
        f.write("# SURVEY.md 8(c) G9 derives the same numbers independently: 1 2 5 9 17 32 61 116 229 460 948 2007\n")
        for lev, n in counts.items():
            f.write("%s %d\n" % (lev, n))


if __name__ == "__main__":
    main()
