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
    """Host logic of the K2 plan (csrc/api.cu plan_jit, csrc/tree_partition.cpp): a table whose register program fits
    an SM runs whole with 256 atoms (threads) per SM; larger ones are cut below the product layer, every
    intermediate cut node lands in exactly one group (checked inside mtp_table_plan) and no program drops below 64
    threads per SM."""
    t = lib.Table(lev)
    plan = t.plan()
    assert plan["partitioned"] == want_part
    if not want_part:
        assert plan["threads_per_sm"] == 256
        return
    assert plan["threads_per_sm"] >= 64
    assert 1 <= plan["groups"] <= 128 and plan["cut_rows"] > plan["groups"]
    assert plan["top_ops"] + plan["ops_below_cut"] == t.n_prod
    assert plan["ops_below_cut"] <= plan["group_ops"] <= 2.0 * plan["ops_below_cut"]      # work duplicated between groups


def _emulate(prog, consts, n_regs, n_slots, inp, n_out, n_bt):
    """Run a K2 register program (csrc/tree_codegen.h K2Op) on numpy columns; NaN marks anything never written."""
    na = inp.shape[1]
    r = np.full((n_regs, na), np.nan)
    sm = np.full((max(n_slots, 1), na), np.nan)
    out = np.full((n_out, na), np.nan)
    bt = np.full((max(n_bt, 1), na), np.nan)
    e = np.zeros(na)
    for op, d, a, b, c, k, x in prog:
        if op == 0: r[d] = inp[x]
        elif op == 2: r[d] = out[x]
        elif op == 3: out[x] = r[a]
        elif op == 4: r[d] = sm[x]
        elif op == 5: sm[x] = r[a]
        elif op == 6: r[d] = r[a] * r[b]
        elif op == 7: r[d] = r[a] * r[b] + r[c]
        elif op == 8: r[d] = consts[k] * r[a]
        elif op == 9: r[d] = consts[k] * r[a] + r[c]
        elif op == 10: r[d] = consts[k]
        elif op == 11: e = e + consts[k] * r[a]
        elif op == 13: bt[x] = r[a]
        elif op == 14: r[d] = r[a] + r[c]
        else: raise AssertionError("unexpected op %d in a whole-table program" % op)
    return e, out, bt


@pytest.mark.parametrize("lev", [6, 10, 16, 20])
def test_k2_register_program_matches_table(lib, lev):
    """The register program the specialised K2 kernel runs (Belady window + spill slots, eager adjoint order) is
    emulated instruction by instruction and compared with the table's plain semantics: forward in list order,
    adjoint by the reverse sweep, E = sum xi B."""
    t = lib.Table(lev)
    rng = np.random.default_rng(100 + lev)
    xi = rng.uniform(-0.1, 0.1, t.n_basis)
    na = 3
    node = np.zeros((t.n_nodes, na))
    node[:t.n_basic] = rng.uniform(-1.2, 1.2, (t.n_basic, na))
    for s0, s1, m, d in t.prod:
        node[d] += m * node[s0] * node[s1]
    E = (xi[:, None] * node[t.basis_node]).sum(axis=0)
    adj = np.zeros_like(node)
    np.add.at(adj, t.basis_node, xi[:, None] * np.ones((1, na)))
    for s0, s1, m, d in t.prod[::-1]:
        w = m * adj[d]
        adj[s0] += w * node[s1]
        adj[s1] += w * node[s0]
    ef = t.k2_program(xi, 0)
    assert ef["prog"][:, 1].max() < ef["n_regs"] and ef["prog"][:, 2].max() < ef["n_regs"]
    e, out, _ = _emulate(ef["prog"], ef["consts"], ef["n_regs"], ef["n_slots"], node[:t.n_basic], t.n_basic, 0)
    scale = np.abs(xi[:, None] * node[t.basis_node]).sum(axis=0) + 1.0
    assert np.all(np.abs(e - E) <= 1e-13 * scale)
    assert not np.isnan(out).any()
    assert np.all(np.abs(out - adj[:t.n_basic]) <= 1e-12 * (1.0 + np.abs(adj[:t.n_basic]).max()))
    vals = t.k2_program(xi, 1)
    _, _, bt = _emulate(vals["prog"], vals["consts"], vals["n_regs"], vals["n_slots"], node[:t.n_basic], t.n_basic, t.n_basis)
    B = node[t.basis_node]
    assert np.all(np.abs(bt - B) <= 1e-13 * (1.0 + np.abs(B)))
