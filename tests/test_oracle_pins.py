"""Pins of the CPU oracle against what the mathematics fixes (SURVEY.md 8(c) pins 1-7).

PAPER.md prints no formula and no value, so every pin is a closed form, an invariant,
a finite difference, a library routine or a brute-force second evaluation.
"""
import itertools
import math

import numpy as np
import pytest
from numpy.polynomial import chebyshev as npcheb

from oracle import basis, mtp
from workloads import random_cluster, make_workload, neighbor_list_bruteforce, reverse_index

R_MIN, R_CUT, NB = 2.0, 5.0, 8
N_MU = {6: 2, 8: 2, 10: 3, 12: 3, 14: 4, 16: 4, 20: 5, 24: 6}


def make_pot(lev, S=1, seed=7, n_beta=NB):
    rng = np.random.default_rng(seed)
    n_mu = N_MU[lev]
    nb = len(basis.basis_functions(lev))
    return mtp.Potential(lev, n_mu, n_beta, R_MIN, R_CUT,
                         rng.uniform(-0.1, 0.1, (S, S, n_mu, n_beta)),
                         rng.uniform(-0.1, 0.1, S), rng.uniform(-0.1, 0.1, nb))


def f_library(pot, zi, zj, r):
    """f_mu(r) through numpy's Chebyshev series routine (independent of the recurrence)."""
    x = (2 * r - pot.r_min - pot.r_cut) / (pot.r_cut - pot.r_min)
    return np.array([npcheb.chebval(x, pot.c[zi][zj][mu]) * (pot.r_cut - r) ** 2
                     for mu in range(pot.n_mu)])


# ---------------------------------------------------------------- pin 6: counts
def test_basis_counts():
    want = {2: 1, 4: 2, 6: 5, 8: 9, 10: 17, 12: 32, 14: 61, 16: 116, 18: 229, 20: 460,
            22: 948, 24: 2007}
    for lev, n in want.items():
        assert len(basis.basis_functions(lev)) == n
    # n_basic = number of unique symmetric components of the moments in use
    for lev, n in {10: 25, 16: 130, 20: 295, 24: 581}.items():
        assert sum((nu + 1) * (nu + 2) // 2 for _, nu in basis.moment_labels(lev)) == n


def test_basis_level10_by_hand():
    """SURVEY.md G9 lists the 17 functions of level <= 10 explicitly."""
    funcs = basis.basis_functions(10)
    names = []
    for f in funcs:
        names.append(tuple(sorted((tuple((mu, nu) for _, mu, nu in lab), ut) for lab, ut in f)))
    m00 = (((0, 0),), ())
    dot11 = (((0, 1), (0, 1)), (1,))
    want = {
        (m00,), (m00, m00), ((((1, 0),), ()),), (dot11,), (m00, m00, m00),
        ((((0, 2), (0, 2)), (2,)),), (m00, (((1, 0),), ())), (m00, dot11), (m00,) * 4,
        ((((2, 0),), ()),), ((((0, 1), (1, 1)), (1,)),), ((((0, 3), (0, 3)), (3,)),),
        ((((0, 1), (0, 1), (0, 2)), (0, 1, 1)),), (m00, (((0, 2), (0, 2)), (2,))),
        (m00, m00, (((1, 0),), ())), (m00, m00, dot11), (m00,) * 5,
    }
    assert set(names) == {tuple(sorted(w)) for w in want}
    assert len(names) == 17


# ---------------------------------------------------------------- radial pins (G1, G5, pin 5)
def test_radial_end_values_and_library():
    Q, dQ = mtp.radial_basis(np.array([R_MIN, R_CUT]), R_MIN, R_CUT, NB)
    for b in range(NB):
        assert Q[b, 0] == pytest.approx((-1) ** b * (R_CUT - R_MIN) ** 2, rel=1e-14)
        assert Q[b, 1] == 0.0 and dQ[b, 1] == 0.0
    r = np.linspace(1.8, 5.0, 41)
    Q, dQ = mtp.radial_basis(r, R_MIN, R_CUT, NB)
    x = (2 * r - R_MIN - R_CUT) / (R_CUT - R_MIN)
    for b in range(NB):
        e = np.zeros(NB)
        e[b] = 1
        assert np.allclose(Q[b], npcheb.chebval(x, e) * (R_CUT - r) ** 2, rtol=1e-13, atol=1e-13)
        # T_b = cos(b arccos x) inside [-1,1]
        ins = np.abs(x) <= 1
        assert np.allclose(Q[b][ins], np.cos(b * np.arccos(x[ins])) * (R_CUT - r[ins]) ** 2, atol=1e-12)
    h = 1e-6
    Qp, _ = mtp.radial_basis(r + h, R_MIN, R_CUT, NB)
    Qm, _ = mtp.radial_basis(r - h, R_MIN, R_CUT, NB)
    assert np.allclose(dQ, (Qp - Qm) / (2 * h), rtol=1e-7, atol=1e-7)


def test_single_radial_function_is_cutoff_parabola():
    """G5: n_beta = 1 => f = c (R_cut - r)^2."""
    pot = make_pot(6, n_beta=1)
    r = np.array([2.3, 3.1, 4.9])
    f, df = mtp.radial_functions(pot, 0, np.zeros(3, int), r)
    for mu in range(pot.n_mu):
        assert np.allclose(f[mu], pot.c[0, 0, mu, 0] * (R_CUT - r) ** 2, rtol=1e-14)
        assert np.allclose(df[mu], -2 * pot.c[0, 0, mu, 0] * (R_CUT - r), rtol=1e-14)


# ---------------------------------------------------------------- pin 1: one neighbour
@pytest.mark.parametrize("lev", [10, 16, 20, 24])
def test_single_neighbour_closed_form(lev):
    """M_{mu,nu} = f_mu(r) r^{(x)nu}  =>  B_alpha = prod_v f_{mu_v}(r) * r^{sum nu}."""
    pot = make_pot(lev, S=2)
    rv = np.array([[1.3, -2.1, 2.4]])
    r = float(np.linalg.norm(rv))
    zi, zj = 1, 0
    f = f_library(pot, zi, zj, r)
    E, B, _ = mtp.atom_eval(pot, zi, rv, np.array([zj]), want_grad=False)
    funcs = basis.basis_functions(lev)
    want = []
    for func in funcs:
        v = 1.0
        for labels, _ in func:
            for (_, mu, nu) in labels:
                v *= f[mu] * r ** nu
        want.append(v)
    want = np.array(want)
    assert np.allclose(B, want, rtol=1e-12, atol=0)
    assert E == pytest.approx(pot.xi0[zi] + pot.xi @ want, rel=1e-12)


# ---------------------------------------------------------------- pin 2: vertex assignment
def dot_form(pot, zi, rv, zj, func):
    """B = prod_components sum_{s: V -> N(i)} prod_v f_{mu_v}(r_{s(v)}) prod_{u<v} (r_su . r_sv)^k."""
    n = rv.shape[0]
    r = np.linalg.norm(rv, axis=1)
    f = np.array([f_library(pot, zi, int(zj[j]), r[j]) for j in range(n)])   # [n][mu]
    dots = rv @ rv.T
    total = 1.0
    for labels, ut in func:
        nv = len(labels)
        acc = 0.0
        for s in itertools.product(range(n), repeat=nv):
            t = 1.0
            for v, (_, mu, nu) in enumerate(labels):
                t *= f[s[v], mu]
            p = 0
            for u in range(nv):
                for v in range(u + 1, nv):
                    if ut[p]:
                        t *= dots[s[u], s[v]] ** ut[p]
                    p += 1
            acc += t
        total *= acc
    return total


@pytest.mark.parametrize("lev,nn", [(10, 4), (12, 4), (16, 3), (20, 3), (24, 2)])
def test_vertex_assignment_brute_force(lev, nn):
    pot = make_pot(lev, S=2, seed=11)
    rng = np.random.default_rng(3)
    rv = rng.uniform(-2.6, 2.6, (nn, 3))
    rv[0] = [1.5, 1.7, -1.9]
    zj = rng.integers(0, 2, nn)
    _, B, _ = mtp.atom_eval(pot, 0, rv, zj, want_grad=False)
    funcs = basis.basis_functions(lev)
    want = np.array([dot_form(pot, 0, rv, zj, fn) for fn in funcs])
    assert np.allclose(B, want, rtol=1e-10, atol=1e-12 * np.abs(want).max())


# ---------------------------------------------------------------- configuration-level pins
def small_config(seed=5, n=14, S=2, box_len=11.0):
    pos, types, box = random_cluster(seed, n, box_len, n_species=S)
    return pos, types, box


def total_energy(pot, pos, types, box, r_list=None, dtype=np.float64):
    off, idx, sh = mtp.brute_force_neighbours(pos, box, pot.r_cut if r_list is None else r_list)
    return mtp.evaluate(pot, pos, types, box, off, idx, sh, dtype=dtype), (off, idx, sh)


@pytest.mark.parametrize("lev", [10, 16, 20, 24])
def test_forces_sum_to_zero_and_match_finite_differences(lev):
    pot = make_pot(lev, S=2)
    pos, types, box = small_config(n={10: 14, 16: 12, 20: 10, 24: 8}[lev])
    out, _ = total_energy(pot, pos, types, box)
    scale = np.abs(out["F"]).max()
    assert np.abs(out["F"].sum(axis=0)).max() <= 1e-11 * scale
    h = 1e-5
    for (k, a) in [(0, 0), (3, 1), (7, 2), (5, 0)]:
        p = pos.copy(); p[k, a] += h
        ep, _ = total_energy(pot, p, types, box)
        p = pos.copy(); p[k, a] -= h
        em, _ = total_energy(pot, p, types, box)
        fd = -(ep["E"] - em["E"]) / (2 * h)
        assert fd == pytest.approx(out["F"][k, a], rel=2e-6, abs=2e-7 * scale)


def test_virial_matches_strain_derivative_and_is_symmetric():
    pot = make_pot(10, S=2)
    pos, types, box = small_config()
    out, _ = total_energy(pot, pos, types, box)
    W = out["W"]
    scale = np.abs(W).max()
    assert np.abs(W - W.T).max() <= 1e-11 * scale
    h = 1e-6
    for (a, b) in [(0, 0), (1, 1), (0, 1), (1, 2)]:
        e = np.zeros((3, 3)); e[a, b] = h
        defp = np.eye(3) + e
        ep, _ = total_energy(pot, pos @ defp.T, types, box @ defp.T)
        defm = np.eye(3) - e
        em, _ = total_energy(pot, pos @ defm.T, types, box @ defm.T)
        fd = -(ep["E"] - em["E"]) / (2 * h)
        assert fd == pytest.approx(W[a, b], rel=5e-6, abs=1e-6 * scale)


def test_rotation_translation_permutation_invariance():
    pot = make_pot(12, S=2)
    pos, types, box = small_config()
    out, _ = total_energy(pot, pos, types, box)
    # rotation (box rotates with the atoms) + translation
    rng = np.random.default_rng(0)
    q, _ = np.linalg.qr(rng.standard_normal((3, 3)))
    if np.linalg.det(q) < 0:
        q[:, 0] *= -1
    pos2 = pos @ q.T + np.array([0.3, -1.2, 2.2]) @ q.T
    box2 = box @ q.T
    out2, _ = total_energy(pot, pos2, types, box2)
    sE = np.abs(out["E_i"]).max()
    assert np.allclose(out2["E_i"], out["E_i"], rtol=0, atol=1e-11 * sE)
    assert np.allclose(out2["B"], out["B"], rtol=1e-9, atol=1e-11 * np.abs(out["B"]).max())
    assert np.allclose(out2["F"], out["F"] @ q.T, rtol=0, atol=1e-10 * np.abs(out["F"]).max())
    # permutation of atoms (same-species swaps included)
    perm = rng.permutation(pos.shape[0])
    out3, _ = total_energy(pot, pos[perm], types[perm], box)
    assert out3["E"] == pytest.approx(out["E"], rel=1e-12)
    assert np.allclose(out3["E_i"], out["E_i"][perm], rtol=0, atol=1e-11 * sE)
    assert np.allclose(out3["F"], out["F"][perm], rtol=0, atol=1e-10 * np.abs(out["F"]).max())


def test_species_relabelling():
    """G6: swapping species labels together with c and xi0 leaves every E_i unchanged;
    c is NOT assumed symmetric, so using c[z_j][z_i] instead must change the result."""
    pot = make_pot(10, S=2)
    pos, types, box = small_config()
    out, _ = total_energy(pot, pos, types, box)
    pot2 = mtp.Potential(pot.lev_max, pot.n_mu, pot.n_beta, pot.r_min, pot.r_cut,
                         pot.c[::-1, ::-1].copy(), pot.xi0[::-1].copy(), pot.xi)
    out2, _ = total_energy(pot2, pos, 1 - types, box)
    assert np.allclose(out2["E_i"], out["E_i"], rtol=1e-13)
    pot3 = mtp.Potential(pot.lev_max, pot.n_mu, pot.n_beta, pot.r_min, pot.r_cut,
                         np.swapaxes(pot.c, 0, 1).copy(), pot.xi0, pot.xi)
    out3, _ = total_energy(pot3, pos, types, box)
    assert not np.allclose(out3["E_i"], out["E_i"], rtol=1e-6)


def test_skin_entries_contribute_nothing_and_cutoff_is_smooth():
    pot = make_pot(10)
    pos, types, box = small_config(S=1)
    out, _ = total_energy(pot, pos, types, box)
    out_skin, (off, idx, sh) = total_energy(pot, pos, types, box, r_list=5.6)
    assert idx.shape[0] > 0
    assert np.array_equal(out_skin["E_i"], out["E_i"])
    assert np.array_equal(out_skin["F"], out["F"])
    # one neighbour moved across R_cut: E changes by O((R_cut - r)^2)
    rv = np.array([[2.2, 0.3, -0.4], [0.0, 0.0, 1.0]])
    vals = []
    for eps in (1e-3, 1e-4, 0.0, -1e-4):
        rv[1] = [0.0, 0.0, R_CUT - eps]
        vals.append(mtp.atom_eval(pot, 0, rv, np.zeros(2, int), want_grad=False)[0])
    assert vals[2] == vals[3]                       # outside: exactly the one-neighbour value
    assert abs(vals[1] - vals[2]) < 1e-6 * max(1.0, abs(vals[2]))
    assert abs(vals[0] - vals[2]) < 1e-4 * max(1.0, abs(vals[2]))


def test_below_rmin_and_empty_neighbourhood():
    """G2: r < R_min is evaluated by the same polynomial (F = -grad E stays exact);
    G20: an atom without neighbours has E_i = xi0[z_i] and no force."""
    pot = make_pot(10)
    rv = np.array([[1.9, 0.0, 0.0], [-1.0, 2.5, 0.7], [0.4, -2.2, 2.9]])
    z = np.zeros(3, int)
    _, _, d = mtp.atom_eval(pot, 0, rv, z)
    h = 1e-6
    for a in range(3):
        p = rv.copy(); p[0, a] += h
        m = rv.copy(); m[0, a] -= h
        fd = (mtp.atom_eval(pot, 0, p, z, want_grad=False)[0]
              - mtp.atom_eval(pot, 0, m, z, want_grad=False)[0]) / (2 * h)
        assert fd == pytest.approx(d[0, a], rel=1e-6, abs=1e-8)
    E, B, d = mtp.atom_eval(pot, 0, np.zeros((0, 3)), np.zeros(0, int))
    assert E == pot.xi0[0] + pot.xi @ B and d.shape == (0, 3)
    # with no neighbours every moment is zero, hence every B
    assert np.all(B == 0.0)


# ---------------------------------------------------------------- pin 7: grades
def test_grade_identities():
    pot = make_pot(10, S=2)
    pos, types, box = small_config(n=20)
    out, _ = total_energy(pot, pos, types, box)
    B = out["B"]
    n_basis = B.shape[1]
    assert np.array_equal(mtp.grade_neighbourhood(B, np.eye(n_basis)), np.abs(B).max(axis=1))
    # active set = rows of B of n_basis chosen atoms => those atoms have gamma = 1
    rows = np.arange(n_basis)
    A = B[rows]
    Ainv = np.linalg.inv(A)
    g = mtp.grade_neighbourhood(B, Ainv)
    assert np.allclose(g[rows], 1.0, rtol=1e-6)
    gc, Bsum = mtp.grade_configuration(B, Ainv)
    assert np.allclose(Bsum, B.sum(axis=0))
    assert gc == pytest.approx(mtp.grade_neighbourhood(Bsum[None, :], Ainv)[0], rel=1e-14)
    # direct loop definition
    k_best = max(abs(sum(B[3, a] * Ainv[a, k] for a in range(n_basis))) for k in range(n_basis))
    assert g[3] == pytest.approx(k_best, rel=1e-12)


def test_long_double_arbiter_agrees():
    """G16: the fp64 oracle and the long-double run agree to fp64 rounding."""
    if np.finfo(np.longdouble).eps >= np.finfo(np.float64).eps:
        pytest.skip("no extended precision on this platform")
    pot = make_pot(16, S=2)
    pos, types, box = small_config(n=10)
    o64, _ = total_energy(pot, pos, types, box)
    o80, _ = total_energy(pot, pos, types, box, dtype=np.longdouble)
    sE = np.abs(o80["E_i"]).max()
    assert float(np.abs(o64["E_i"] - o80["E_i"]).max()) < 1e-12 * float(sE)
    assert float(np.abs(o64["F"] - o80["F"]).max()) < 1e-11 * float(np.abs(o80["F"]).max())


# ---------------------------------------------------------------- step 1: pair vectors and neighbour lists
def _sheared_box():
    """A triclinic box (rows = lattice vectors) whose three heights all exceed 2 R_cut."""
    box = np.array([[12.5, 0.0, 0.0], [3.1, 12.0, 0.0], [-2.2, 1.7, 11.6]])
    vol = abs(np.linalg.det(box))
    heights = [vol / np.linalg.norm(np.cross(box[(k + 1) % 3], box[(k + 2) % 3])) for k in range(3)]
    assert min(heights) > 2 * R_CUT
    return box


@pytest.mark.parametrize("triclinic", [False, True])
def test_minimum_image_branch_equals_explicit_shifts(triclinic):
    """pair_vectors(shift=None) (G17: minimum image, legal when every box height exceeds 2 R_cut) must give exactly
    the vectors of the explicit-shift branch for every listed pair, in an orthorhombic and in a sheared box."""
    rng = np.random.default_rng(17)
    if triclinic:
        box = _sheared_box()
        pos = rng.uniform(0, 1, (26, 3)) @ box
    else:
        pos, _, box = random_cluster(9, 24, 11.0)
    off, idx, sh = mtp.brute_force_neighbours(pos, box, R_CUT)
    assert idx.shape[0] > 50 and np.abs(sh).max() == 1          # pairs through the periodic boundary are present
    for i in range(pos.shape[0]):
        js_a, rv_a = mtp.pair_vectors(i, pos, box, off, idx, sh)
        js_b, rv_b = mtp.pair_vectors(i, pos, box, off, idx, None)
        assert np.array_equal(js_a, js_b)
        assert np.allclose(rv_a, rv_b, rtol=0, atol=1e-12)
        assert np.all(np.linalg.norm(rv_a, axis=1) < R_CUT)
    # and the brute-force list itself: every pair within R_cut of the 27 images is listed exactly once, nothing else
    n = pos.shape[0]
    count = 0
    for i in range(n):
        for j in range(n):
            for s in itertools.product((-1, 0, 1), repeat=3):
                if i == j and s == (0, 0, 0):
                    continue
                v = pos[j] - pos[i] + np.array(s) @ box
                count += bool(v @ v < R_CUT * R_CUT)
    assert count == idx.shape[0]


def test_sheared_box_energy_is_rotation_invariant_and_forces_match_fd():
    """The triclinic path of the oracle (shift . box with a non-diagonal box) against invariance and finite differences."""
    pot = make_pot(10, S=2)
    rng = np.random.default_rng(23)
    box = _sheared_box()
    pos = rng.uniform(0, 1, (16, 3)) @ box
    types = rng.integers(0, 2, 16).astype(np.int32)
    out, (off, idx, sh) = total_energy(pot, pos, types, box)
    out_mi = mtp.evaluate(pot, pos, types, box, off, idx, None)
    assert np.allclose(out_mi["E_i"], out["E_i"], rtol=1e-13) and np.allclose(out_mi["F"], out["F"], rtol=0, atol=1e-12 * np.abs(out["F"]).max())
    q, _ = np.linalg.qr(rng.standard_normal((3, 3)))
    out2, _ = total_energy(pot, pos @ q.T, types, box @ q.T)
    assert np.allclose(out2["E_i"], out["E_i"], rtol=0, atol=1e-11 * np.abs(out["E_i"]).max())
    h = 1e-5
    for (k, a) in [(2, 0), (9, 2)]:
        p = pos.copy(); p[k, a] += h
        ep, _ = total_energy(pot, p, types, box)
        p = pos.copy(); p[k, a] -= h
        em, _ = total_energy(pot, p, types, box)
        assert -(ep["E"] - em["E"]) / (2 * h) == pytest.approx(out["F"][k, a], rel=2e-6, abs=2e-7 * np.abs(out["F"]).max())


@pytest.mark.parametrize("ci", [0, 1])
def test_three_neighbour_list_builders_agree(ci):
    """BASELINE.json configs[0] and configs[1] at full size: the lattice-stencil list the workloads use (both arms
    consume it) equals the vectorised brute-force 27-image search bit for bit (off, idx, shift), and the oracle's
    own pure-Python brute force equals both (every row at 128 atoms, sampled rows at 2 000 atoms); the reverse index
    is an involution that maps (i, j, s) to (j, i, -s)."""
    w = make_workload(ci, 1, with_rev=True)
    assert w.n_atoms == (128, 2000)[ci]
    off, idx, sh = neighbor_list_bruteforce(w.pos, w.box, R_CUT)
    assert np.array_equal(off, w.off) and np.array_equal(idx, w.idx) and np.array_equal(sh, w.shift)
    rows = list(range(w.n_atoms)) if ci == 0 else [0, 1, 77, 512, 999, 1203, 1998, 1999]
    o_off, o_idx, o_sh = mtp.brute_force_neighbours(w.pos, w.box, R_CUT, rows=rows)
    for q, i in enumerate(rows):
        a, b = w.off[i], w.off[i + 1]
        assert np.array_equal(o_idx[o_off[q]:o_off[q + 1]], w.idx[a:b])
        assert np.array_equal(o_sh[o_off[q]:o_off[q + 1]], w.shift[a:b])
    rev = w.rev
    i_of = np.repeat(np.arange(w.n_atoms), np.diff(w.off))
    assert np.array_equal(rev[rev], np.arange(w.nnz))
    assert np.array_equal(w.idx[rev], i_of) and np.array_equal(i_of[rev], w.idx)
    assert np.array_equal(w.shift[rev], -w.shift)
    assert np.array_equal(reverse_index(w.off, w.idx, w.shift), rev)
