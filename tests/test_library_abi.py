"""-m "not gpu": the C-ABI library loads, exports every symbol include/mtp_b200.h declares,
and its host-side basis enumerator agrees with the oracle's independent enumeration."""
import ctypes
import re
import os

import numpy as np
import pytest

from oracle import basis as obasis
from oracle import mtp as omtp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_exports_match_header(lib):
    hdr = open(os.path.join(ROOT, "include", "mtp_b200.h")).read()
    declared = set(re.findall(r"\b(mtp_[a-z_0-9]+)\s*\(", hdr))
    assert declared == set(lib.EXPORTS)
    so = ctypes.CDLL(lib.LIB_PATH)
    for name in declared:
        assert hasattr(so, name), name


@pytest.mark.parametrize("lev", [2, 4, 6, 8, 10, 12, 14, 16, 18, 20, 22, 24])
def test_enumerator_order_matches_oracle(lib, lev):
    """G11: both sides implement the canonical order independently; the lists must be identical."""
    t = lib.Table(lev)
    funcs = obasis.basis_functions(lev)
    assert t.n_basis == len(funcs)
    for a, f in enumerate(funcs):
        assert t.describe(a) == obasis.describe(f)
    labels = obasis.moment_labels(lev)
    assert t.n_basic == sum((nu + 1) * (nu + 2) // 2 for _, nu in labels)
    assert t.n_mu == 1 + max(mu for mu, _ in labels)


@pytest.mark.parametrize("lev", [10, 16, 20])
def test_contraction_table_reproduces_oracle_basis(lib, lev):
    """Interpret the emitted table on the CPU with the oracle's dense moments as input."""
    t = lib.Table(lev)
    rng = np.random.default_rng(lev)
    pot = omtp.Potential(lev, t.n_mu, 8, 2.0, 5.0, rng.uniform(-0.1, 0.1, (1, 1, t.n_mu, 8)), np.zeros(1),
                         np.zeros(t.n_basis))
    rv = rng.uniform(-2.6, 2.6, (9, 3))
    f, _ = omtp.radial_functions(pot, 0, np.zeros(9, int), np.linalg.norm(rv, axis=1))
    M, _ = omtp.moments(pot, f, rv)
    B, _ = omtp.basis_values(pot, M)
    node = np.zeros(t.n_nodes)
    for k, (mu, a, b, c) in enumerate(t.basic):
        node[k] = M[(mu, a + b + c)][(0,) * a + (1,) * b + (2,) * c]
    for s0, s1, m, d in t.prod:
        node[d] += m * node[s0] * node[s1]
    got = node[t.basis_node]
    assert np.allclose(got, B, rtol=1e-11, atol=1e-13 * np.abs(B).max())


def test_no_device_means_error_not_fallback(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    t = lib.Table(6)
    with pytest.raises(lib.MtpError) as e:
        lib.Potential(t, 1, 8, 2.0, 5.0, np.zeros((1, 1, t.n_mu, 8)), np.zeros(1), np.zeros(t.n_basis))
    assert e.value.code == lib.ECUDA


@pytest.mark.parametrize("lev,want_part", [(10, 0), (16, 0), (20, 1), (24, 1)])
def test_table_plan_partitions_only_large_tables(lib, lev, want_part):
    """Host logic of the K2 partition (csrc/tree_partition.cpp): small tables run whole with 64 atoms per CTA; large
    ones are cut, every intermediate cut node lands in exactly one group (checked inside mtp_table_plan), all groups fit
    at least 32 atoms per CTA, and the duplicated work stays moderate."""
    plan = lib.Table(lev).plan()
    assert plan["partitioned"] == want_part
    if not want_part:
        assert plan["atoms_per_cta"] == 64
        return
    assert plan["atoms_per_cta"] < 32 and plan["group_atoms_per_cta"] >= 32
    assert 1 <= plan["groups"] <= 24 and plan["cut_rows"] > plan["groups"]
    assert plan["top_ops"] + plan["ops_below_cut"] == lib.Table(lev).n_prod
    assert plan["ops_below_cut"] <= plan["group_ops"] <= 1.5 * plan["ops_below_cut"]
