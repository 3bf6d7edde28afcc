"""CPU oracle for the Moment Tensor Potential hot path -- TEST INFRASTRUCTURE ONLY.

Plain, slow, obviously-correct numpy (fp64 by default, x87 long double as the
rounding arbiter) written from BASELINE.json `north_star` / SURVEY.md 8(c) steps 1-8
(PAPER.md states no formula).  It shares no code with the
CUDA path in `paper_2510_00193_b200/` and neither imports the other.  Only `tests/`,
`__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference` legs may
import it; the product path never does.

Pins (tests/test_oracle_*.py, all `-m "not gpu"`): single-neighbour closed form,
vertex-assignment (dot-product) brute force, rotation / translation / permutation
invariance, sum(F)=0, F=-grad E and virial=-dE/d(strain) by central differences,
smooth vanishing at R_cut, basis counts 1,2,5,9,17,32,61,116,229,460,948,2007,
grade identities.  Parity against MLIP-3 / LAMMPS output for a trained potential is
"parity unpinned": no such output or potential file exists in this environment.
"""
