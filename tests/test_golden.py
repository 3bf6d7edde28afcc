"""Stored expected values (tests/golden/, written by make_golden.py from oracle/ only): the oracle must
reproduce them (CPU), and the CUDA path must match them through the C ABI (-m gpu)."""
import json
import os

import numpy as np
import pytest

from oracle import basis, mtp
from workloads import random_cluster, Workload, reverse_index

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def load_cases():
    return json.load(open(os.path.join(GOLD, "cluster_cases.json")))["cases"]


def rebuild(case):
    pos, types, box = random_cluster(case["seed"], case["n_atoms"], 11.0, n_species=case["n_species"])
    off, idx, shift = mtp.brute_force_neighbours(pos, box, 5.0)
    rng = np.random.default_rng(case["seed"] + 1)
    S, n_mu = case["n_species"], case["n_mu"]
    nb = len(basis.basis_functions(case["lev"]))
    c = rng.uniform(-0.1, 0.1, (S, S, n_mu, 8))
    xi0 = rng.uniform(-0.1, 0.1, S)
    xi = rng.uniform(-0.1, 0.1, nb)
    return Workload(name="golden", lev_max=case["lev"], n_mu=n_mu, n_beta=8, r_min=2.0, r_cut=5.0, n_species=S, box=box,
                    pos=pos, types=types, c=c, xi0=xi0, xi=xi, off=off, idx=idx, shift=shift,
                    rev=reverse_index(off, idx, shift))


def test_basis_counts_file():
    for line in open(os.path.join(GOLD, "basis_counts.txt")):
        if line.startswith("#"):
            continue
        lev, n = map(int, line.split())
        assert len(basis.basis_functions(lev)) == n


@pytest.mark.parametrize("k", [0, 1])
def test_oracle_reproduces_golden(k):
    case = load_cases()[k]
    w = rebuild(case)
    assert w.nnz == case["nnz"]
    pot = mtp.Potential(w.lev_max, w.n_mu, 8, 2.0, 5.0, w.c, w.xi0, w.xi)
    out = mtp.evaluate(pot, w.pos, w.types, w.box, w.off, w.idx, w.shift)
    assert np.allclose(out["E_i"], case["E_i"], rtol=1e-12, atol=1e-12 * np.abs(case["E_i"]).max())
    assert np.allclose(out["F"], case["F"], rtol=1e-10, atol=1e-10 * np.abs(case["F"]).max())
    assert np.allclose(mtp.virial6(out["W"]), case["virial"], rtol=1e-10, atol=1e-10 * np.abs(case["virial"]).max())


@pytest.mark.gpu
@pytest.mark.parametrize("k", [0, 1])
def test_gpu_matches_golden(lib, k):
    import torch
    from _util import gpu_pot, to_dev
    case = load_cases()[k]
    w = rebuild(case)
    pot = gpu_pot(lib, w)
    d = to_dev(w, torch)
    out = pot.compute(d["pos"], d["types"], w.box, d["off"], d["idx"], d["shift"], d["rev"])
    torch.cuda.synchronize()
    Ei, F = out["Ei"].cpu().numpy(), out["F"].cpu().numpy()
    # the stated tolerances, with the scales of the summed terms taken from an oracle run
    from _util import oracle_pot, scales
    opot = oracle_pot(w)
    ref = mtp.evaluate(opot, w.pos, w.types, w.box, w.off, w.idx, w.shift)
    sE, sF = scales(opot, ref, w.off, w.idx)
    assert np.all(np.abs(Ei - np.asarray(case["E_i"])) <= 1e-10 * sE)
    assert np.all(np.abs(F - np.asarray(case["F"])) <= 1e-9 * sF[:, None])
    rv = np.concatenate([mtp.pair_vectors(i, w.pos, w.box, w.off, w.idx, w.shift)[1] for i in range(w.n_atoms)])
    sW = max(1.0, np.abs(rv[:, :, None] * ref["d"][:, None, :]).sum())
    assert np.all(np.abs(out["virial"].cpu().numpy() - np.asarray(case["virial"])) <= 1e-10 * sW)
    pot.close()
