"""-m gpu: the device neighbour list (bit-exact against the brute-force searches), the positions-only host path and
the velocity-Verlet loop, all through the C ABI."""
import numpy as np
import pytest

from oracle import mtp as omtp
from workloads import make_workload, neighbor_list_bruteforce, reverse_index
from _util import n_basis_of, gpu_pot, to_dev

pytestmark = pytest.mark.gpu
KFTM2V = 1.602176634e-19 / 1.66053906660e-27 * 1e-4      # eV/A / (g/mol) -> A/ps^2


@pytest.fixture(scope="module")
def torch():
    import torch as t
    assert t.cuda.is_available()
    return t


def build(lib, torch, pos, box, r, **kw):
    nb = lib.neighbors_build(torch.as_tensor(np.ascontiguousarray(pos)).cuda(), box, r, **kw)
    n = nb["nnz"]
    return (nb["off"].cpu().numpy(), nb["idx"].cpu().numpy()[:n], nb["shift"].cpu().numpy()[:n],
            nb["rev"].cpu().numpy()[:n] if nb["rev"] is not None else None, nb)


@pytest.mark.parametrize("ci", [0, 1])
def test_list_is_bit_exact_at_configs_1_and_2(lib, torch, ci):
    """Integer work: off / idx / shift / rev equal the brute-force 27-image search bit for bit (the oracle's own search on
    every row at 128 atoms and on sampled rows at 2 000 atoms; the vectorised brute force on every row)."""
    w = make_workload(ci, 1)
    off, idx, sh, rev, nb = build(lib, torch, w.pos, w.box, 5.0)
    assert nb["errors"] == 0 and nb["nnz"] == w.nnz
    b_off, b_idx, b_sh = neighbor_list_bruteforce(w.pos, w.box, 5.0)
    assert np.array_equal(off, b_off) and np.array_equal(idx, b_idx) and np.array_equal(sh, b_sh)
    rows = list(range(w.n_atoms)) if ci == 0 else [0, 3, 500, 1234, 1999]
    o_off, o_idx, o_sh = omtp.brute_force_neighbours(w.pos, w.box, 5.0, rows=rows)
    for q, i in enumerate(rows):
        assert np.array_equal(o_idx[o_off[q]:o_off[q + 1]], idx[off[i]:off[i + 1]])
        assert np.array_equal(o_sh[o_off[q]:o_off[q + 1]], sh[off[i]:off[i + 1]])
    assert np.array_equal(rev, reverse_index(b_off, b_idx, b_sh))


def test_sheared_small_and_unwrapped_boxes(lib, torch):
    """Triclinic box; a box with fewer than three cells per direction and one with a single cell (the same cell is
    reached through several images); atoms given outside the box."""
    rng = np.random.default_rng(7)
    box = np.array([[12.5, 0.0, 0.0], [3.1, 12.0, 0.0], [-2.2, 1.7, 11.6]])
    pos = rng.uniform(0, 1, (60, 3)) @ box
    for bx, ps, r in [(box, pos, 5.0), (np.eye(3) * 11.0, rng.uniform(0, 11.0, (50, 3)), 5.0),
                      (np.eye(3) * 7.0, rng.uniform(0, 7.0, (20, 3)), 5.0)]:
        off, idx, sh, rev, nb = build(lib, torch, ps, bx, r)
        o_off, o_idx, o_sh = omtp.brute_force_neighbours(ps, bx, r)
        assert nb["errors"] == 0
        assert np.array_equal(off, o_off) and np.array_equal(idx, o_idx) and np.array_equal(sh, o_sh)
        assert np.array_equal(rev, reverse_index(o_off, o_idx, o_sh))
    # atoms shifted out of the box by one lattice vector: the definition's pairs for the given coordinates
    ps = pos.copy()
    ps[::3] += box[0]
    ps[1::5] -= box[2]
    off, idx, sh, rev, nb = build(lib, torch, ps, box, 5.0)
    o_off, o_idx, o_sh = omtp.brute_force_neighbours(ps, box, 5.0)       # images in {-1,0,1}^3 of the GIVEN coordinates
    assert np.array_equal(off, o_off) and np.array_equal(idx, o_idx) and np.array_equal(sh, o_sh)
    assert o_idx.shape[0] < omtp.brute_force_neighbours(pos, box, 5.0)[1].shape[0]     # some pairs would need a shift of 2


def test_capacity_and_count_only(lib, torch):
    w = make_workload(0, 1)
    pos = torch.as_tensor(w.pos).cuda()
    nb = lib.neighbors_build(pos, w.box, 5.0, capacity=0)
    assert nb["nnz"] == w.nnz and np.array_equal(nb["off"].cpu().numpy(), w.off)
    for want_rev in (True, False):                                      # truncated: the count still says what is needed,
        nb = lib.neighbors_build(pos, w.box, 5.0, capacity=1000, want_rev=want_rev)   # the first `capacity` pairs are there
        assert nb["nnz"] == w.nnz
        assert np.array_equal(nb["idx"].cpu().numpy()[:1000], w.idx[:1000])
        assert np.array_equal(nb["shift"].cpu().numpy()[:1000], w.shift[:1000])
    nb = lib.neighbors_build(pos, w.box, 5.0, want_rev=False)           # the two-search form (no rev array to stash rows in)
    assert nb["nnz"] == w.nnz and np.array_equal(nb["idx"].cpu().numpy()[:w.nnz], w.idx)
    assert np.array_equal(nb["shift"].cpu().numpy()[:w.nnz], w.shift)


def test_config4_sampled_rows(lib, torch):
    """BASELINE.json configs[3] at full size: the device list has the workload's pair count and its rows equal the
    stencil list's (pinned against brute force on the CPU) on sampled rows; rev is an involution."""
    w = make_workload(3, 1)
    off, idx, sh, rev, nb = build(lib, torch, w.pos, w.box, 5.0)
    assert nb["errors"] == 0 and nb["nnz"] == w.nnz and np.array_equal(off, w.off)
    rng = np.random.default_rng(1)
    for i in rng.choice(w.n_atoms, 200, replace=False):
        a, b = off[i], off[i + 1]
        assert np.array_equal(idx[a:b], w.idx[a:b]) and np.array_equal(sh[a:b], w.shift[a:b])
    p = rng.choice(w.nnz, 100000, replace=False)
    assert np.array_equal(rev[rev[p]], p) and np.array_equal(rev[p], w.rev[p])


def test_host_positions_path_equals_host_list_path(lib, torch):
    w = make_workload(1, n_basis_of(16), cells=5)
    pot = gpu_pot(lib, w)
    pot.set_option(lib.OPT_FORCE_MODE, lib.FORCE_GATHER)
    a = pot.compute_host(w.pos, w.types, w.box, w.off, w.idx, w.shift, w.rev)
    b = pot.compute_host_pos(w.pos, w.types, w.box)
    assert b["nnz"] == w.nnz
    for k in ("E", "Ei", "F", "virial"):
        assert np.array_equal(a[k], b[k]), k
    c = pot.compute_host_pos(w.pos, w.types, w.box)                     # second call: buffers already sized
    assert np.array_equal(b["F"], c["F"])
    pot.close()


def test_coordinates_that_are_not_finite_are_counted_not_followed(lib, torch):
    """An MD run that blew up hands the list build NaN / inf / 1e300: no fault, d_info[1] counts them, the other atoms'
    rows are those of the brute-force search without the bad atoms' pairs."""
    w = make_workload(0, 1)
    pos = w.pos.copy()
    bad = [3, 40, 77]
    pos[3, 0] = np.nan; pos[40, 1] = np.inf; pos[77, 2] = -1e300
    off, idx, sh, rev, nb = build(lib, torch, pos, w.box, 5.0)
    assert nb["errors"] == 3
    b_off, b_idx, b_sh = neighbor_list_bruteforce(w.pos, w.box, 5.0)
    for i in range(w.n_atoms):
        keep = ~np.isin(b_idx[b_off[i]:b_off[i + 1]], bad)
        want = b_idx[b_off[i]:b_off[i + 1]][keep] if i not in bad else np.zeros(0, dtype=np.int32)
        assert np.array_equal(idx[off[i]:off[i + 1]], want), i


def test_velocity_verlet_loop(lib, torch):
    """mtp_md_run: (1) zero steps = one force evaluation; (2) two steps equal the same update written out in numpy on
    top of mtp_compute's forces; (3) over 200 steps the total energy drifts by a small fraction of the kinetic energy,
    with list rebuilds every 10 steps at a 1 A skin giving the same trajectory as rebuilding every step.  (The seeded
    random coefficients make a stiff, unphysical potential -- forces of 1e3 - 1e4 eV/A at level 10 -- hence steps of 0.01 and 0.001 fs.)"""
    w = make_workload(0, n_basis_of(10))
    pot = gpu_pot(lib, w)
    d = to_dev(w, torch)
    rng = np.random.default_rng(3)
    mass = np.array([55.845])
    vel0 = rng.normal(0.0, 2.0, (w.n_atoms, 3))                         # A/ps
    vel0 -= vel0.mean(axis=0)
    cap = int(w.nnz * 1.6)
    ref = pot.compute(d["pos"], d["types"], w.box, d["off"], d["idx"], d["shift"], d["rev"])
    torch.cuda.synchronize()
    pos, vel = d["pos"].clone(), torch.as_tensor(vel0).cuda()
    out = pot.md_run(pos, vel, d["types"], w.box, mass, 1e-5, 0, 1, 0.0, cap)
    torch.cuda.synchronize()
    assert np.array_equal(out["F"].cpu().numpy(), ref["F"].cpu().numpy()) and np.array_equal(pos.cpu().numpy(), w.pos)
    ke0 = 0.5 / KFTM2V * (mass[0] * vel0 ** 2).sum()
    assert out["E"].cpu().numpy()[1] == pytest.approx(ke0, rel=1e-13)
    # (2) two steps by hand
    dt = 1e-5
    x, v, F = w.pos.copy(), vel0.copy(), ref["F"].cpu().numpy()
    for _ in range(2):
        v = v + 0.5 * dt * KFTM2V / mass[0] * F
        x = x + dt * v
        nb = lib.neighbors_build(torch.as_tensor(x).cuda(), w.box, 5.0)
        o = pot.compute(torch.as_tensor(x).cuda(), d["types"], w.box, nb["off"], nb["idx"][:nb["nnz"]], nb["shift"][:nb["nnz"]],
                        nb["rev"][:nb["nnz"]])
        torch.cuda.synchronize()
        F = o["F"].cpu().numpy()
        v = v + 0.5 * dt * KFTM2V / mass[0] * F
    pos, vel = d["pos"].clone(), torch.as_tensor(vel0).cuda()
    out = pot.md_run(pos, vel, d["types"], w.box, mass, dt, 2, 1, 0.0, cap)
    torch.cuda.synchronize()
    L = w.box[0, 0]
    dx = pos.cpu().numpy() - x
    dx -= np.round(dx / L) * L                                          # md_run wraps atoms into the box at a rebuild
    assert np.abs(dx).max() < 1e-12 and np.abs(vel.cpu().numpy() - v).max() < 1e-10
    # (3) energy conservation and rebuild cadence
    res = {}
    dt = 1e-6
    for every, skin in ((1, 0.0), (10, 1.0)):
        pos, vel = d["pos"].clone(), torch.as_tensor(vel0).cuda()
        o = pot.md_run(pos, vel, d["types"], w.box, mass, dt, 200, every, skin, int(w.nnz * 2.2))
        torch.cuda.synchronize()
        info = o["info"].cpu().numpy()
        assert info[1] == 0 and info[0] <= int(w.nnz * 2.2)
        assert pot.get_option(lib.INFO_INPUT_ERRORS) == 0 and pot.get_option(lib.INFO_SCRATCH_OVERFLOW) == 0
        res[every] = (o["E"].cpu().numpy().copy(), pos.cpu().numpy().copy())
    e0 = ref["E"].cpu().numpy()[0] + ke0
    e1 = res[1][0].sum()
    assert res[1][0][1] > 2 * ke0                                        # the atoms did pick up kinetic energy
    assert abs(e1 - e0) < 1e-3 * (res[1][0][1] + ke0)
    dx = res[1][1] - res[10][1]
    dx -= np.round(dx / L) * L
    assert np.abs(dx).max() < 1e-9 and abs(res[1][0].sum() - res[10][0].sum()) < 1e-9 * abs(e0)
    pot.close()


def test_md_loop_with_grade_policy(lib, torch):
    """mtp_md_run_al: grades on the initial configuration and after every 5th step.
    Expected values come from the pieces already tested: the trajectory of mtp_md_run stopped at the same steps, the
    grades of mtp_grade on it.  Checked: the per-evaluation maximum (device reduction) bit for bit, which steps are
    kept and their positions, the break."""
    w = make_workload(0, n_basis_of(10), with_ainv=True)
    pot = gpu_pot(lib, w)
    d = to_dev(w, torch)
    Ainv = torch.as_tensor(w.Ainv).cuda()
    rng = np.random.default_rng(5)
    mass = np.array([55.845])
    vel0 = rng.normal(0.0, 2.0, (w.n_atoms, 3))
    cap, dt, every, skin, X, steps = int(w.nnz * 2.2), 1e-6, 10, 1.0, 5, 20
    # reference: run to step s with the plain loop, then grade that configuration on that list
    want = {}
    for s in range(0, steps + 1, X):
        pos, vel = d["pos"].clone(), torch.as_tensor(vel0).cuda()
        pot.md_run(pos, vel, d["types"], w.box, mass, dt, s, every, skin, cap)
        # the list the loop holds at step s: built at the last multiple of `every` (positions wrapped there)
        p2, v2 = d["pos"].clone(), torch.as_tensor(vel0).cuda()
        pot.md_run(p2, v2, d["types"], w.box, mass, dt, (s // every) * every, every, skin, cap)
        nb = lib.neighbors_build(p2, w.box, 5.0 + skin)
        n = nb["nnz"]
        g = pot.grade(pos, d["types"], w.box, nb["off"], nb["idx"][:n], Ainv, nb["shift"][:n], mode=2)
        torch.cuda.synchronize()
        want[s] = (pos.cpu().numpy(), float(g["gamma_atom"].max()), float(g["gamma_cfg"][0]), g["gamma_atom"].cpu().numpy())
    for mode in (0, 1):
        grades = [want[s][1 + mode] for s in sorted(want)]
        thr = 0.5 * (min(grades) + max(grades))
        assert min(grades) < thr < max(grades)
        pos, vel = d["pos"].clone(), torch.as_tensor(vel0).cuda()
        o = pot.md_run_al(pos, vel, d["types"], w.box, mass, dt, steps, every, skin, cap, Ainv, X, mode, thr, 1e300, 16)
        torch.cuda.synchronize()
        keep = [s for s in sorted(want) if want[s][1 + mode] > thr]
        assert o["steps_done"] == steps and not o["stopped"] and o["n_evaluations"] == steps // X + 1
        assert o["sel_step"] == keep and o["sel_grade"] == [want[s][1 + mode] for s in keep]
        assert o["max_grade"] == max(grades)
        for k, s in enumerate(keep):
            assert np.array_equal(o["selected"][k].cpu().numpy(), want[s][0])
        if mode == 0:                                                    # the dump of the kept configurations reads back exactly
            import os, tempfile
            path = os.path.join(tempfile.mkdtemp(), "selected.xyz")
            assert lib.dump_selected(path, o, d["types"], w.box) == len(keep)
            lines = open(path).read().split("\n")
            assert len(lines) == len(keep) * (w.n_atoms + 2) + 1 and ("step=%d " % keep[0]) in lines[1]
            back = np.array([[float(v) for v in ln.split()[1:]] for ln in lines[2:2 + w.n_atoms]])
            assert np.array_equal(back, want[keep[0]][0])
        if mode == 0:
            assert np.array_equal(o["gamma_atom"].cpu().numpy(), want[steps][3])
        assert np.array_equal(pos.cpu().numpy(), want[steps][0])
        # at most two kept; break at the first evaluation above the threshold
        pos, vel = d["pos"].clone(), torch.as_tensor(vel0).cuda()
        o = pot.md_run_al(pos, vel, d["types"], w.box, mass, dt, steps, every, skin, cap, Ainv, X, mode, -1.0, thr, 2)
        assert o["stopped"] and o["steps_done"] == keep[0] and o["sel_step"] == [0, X][:o["n_evaluations"]][:2]
        assert np.array_equal(pos.cpu().numpy(), want[keep[0]][0])
    pot.close()


def test_skin_list_rows_are_compacted_not_multiplied_by_zero(lib, torch):
    """MTP_OPT_SKIN_LIST: a list built at R_cut + 1 A through the large-system kernels, with the rows compacted to the
    entries within R_cut, equals the same list evaluated with the skin pairs multiplied by zero, and the list built at
    R_cut itself: E_i bit for bit (the kept entries come in the same order, and adding zeros changes no sum); forces and
    virial to rounding (an atom's own pairs are summed by TN threads according to their position in the row, which the
    dropped entries shift).  Several chunks, explicit shifts and minimum image, both force modes."""
    w = make_workload(3, n_basis_of(16), cells=8)
    pot = gpu_pot(lib, w)
    pot.set_option(lib.OPT_VARIANT, lib.VARIANT_THREAD)
    pot.set_option(lib.OPT_CHUNK_ATOMS, 600)
    pos, types = torch.as_tensor(w.pos).cuda(), torch.as_tensor(w.types).cuda()
    exact, skin = lib.neighbors_build(pos, w.box, 5.0), lib.neighbors_build(pos, w.box, 6.0)
    assert skin["nnz"] > 1.5 * exact["nnz"]

    def run(nb, live, mode, with_shift=True):
        pot.set_option(lib.OPT_SKIN_LIST, live)
        pot.set_option(lib.OPT_FORCE_MODE, mode)
        n = nb["nnz"]
        o = pot.compute(pos, types, w.box, nb["off"], nb["idx"][:n], nb["shift"][:n] if with_shift else None, nb["rev"][:n])
        torch.cuda.synchronize()
        assert pot.get_option(lib.INFO_INPUT_ERRORS) == 0 and pot.get_option(lib.INFO_SCRATCH_OVERFLOW) == 0
        return {k: v.cpu().numpy() for k, v in o.items()}

    for with_shift, chunk in ((True, 600), (False, 600), (True, 0)):       # several chunks, and the automatic single chunk
        pot.set_option(lib.OPT_CHUNK_ATOMS, chunk)
        ref = run(exact, 0, lib.FORCE_GATHER, with_shift)
        zero = run(skin, 0, lib.FORCE_GATHER, with_shift)
        live = run(skin, 1, lib.FORCE_GATHER, with_shift)
        for k in ("E", "Ei"):
            assert np.array_equal(live[k], zero[k]) and np.array_equal(live[k], ref[k]), (k, with_shift)
        for k in ("F", "virial"):
            scale = np.abs(ref[k]).max()
            assert np.abs(live[k] - ref[k]).max() <= 1e-12 * scale and np.abs(zero[k] - ref[k]).max() <= 1e-12 * scale, (k, with_shift)
        again = run(skin, 1, lib.FORCE_GATHER, with_shift)
        assert np.array_equal(again["F"], live["F"])                      # still deterministic
        atom = run(skin, 1, lib.FORCE_ATOMIC, with_shift)
        assert np.array_equal(atom["Ei"], ref["Ei"])
        assert np.abs(atom["F"] - ref["F"]).max() <= 1e-12 * np.abs(ref["F"]).max()
    pot.close()


def test_list_and_md_edge_cases(lib, torch):
    """One atom (its own images only), two atoms out of range (no pairs at all), an atom count that is not a multiple
    of anything, a zero-step MD call on a system without pairs."""
    box = np.eye(3) * 12.0
    one = np.array([[1.0, 2.0, 3.0]])
    off, idx, sh, rev, nb = build(lib, torch, one, box, 5.0)
    assert nb["nnz"] == 0 and off.tolist() == [0, 0] and nb["errors"] == 0
    off, idx, sh, rev, nb = build(lib, torch, one, np.eye(3) * 4.0, 5.0)          # box smaller than the radius: 6 own images at 4 A
    o_off, o_idx, o_sh = omtp.brute_force_neighbours(one, np.eye(3) * 4.0, 5.0)
    assert nb["nnz"] == o_off[-1] == 6 and np.array_equal(sh, o_sh) and np.array_equal(rev, reverse_index(o_off, o_idx, o_sh))
    two = np.array([[1.0, 1.0, 1.0], [7.0, 7.0, 7.0]])
    off, idx, sh, rev, nb = build(lib, torch, two, box, 5.0)
    assert nb["nnz"] == 0 and off.tolist() == [0, 0, 0]
    rng = np.random.default_rng(2)
    pos = rng.uniform(0, 12.0, (37, 3))
    off, idx, sh, rev, nb = build(lib, torch, pos, box, 5.0)
    o_off, o_idx, o_sh = omtp.brute_force_neighbours(pos, box, 5.0)
    assert np.array_equal(off, o_off) and np.array_equal(idx, o_idx) and np.array_equal(sh, o_sh)
    # MD on the pairless system: E = sum xi0, F = 0, nothing moves without velocities
    w = make_workload(0, n_basis_of(10))
    pot = gpu_pot(lib, w)
    p, v, t = torch.as_tensor(two).cuda(), torch.zeros((2, 3), dtype=torch.float64, device="cuda"), torch.zeros(2, dtype=torch.int32, device="cuda")
    o = pot.md_run(p, v, t, box, np.array([55.845]), 1e-3, 3, 1, 0.5, 16)
    torch.cuda.synchronize()
    assert o["info"].cpu().tolist() == [0, 0] and not o["F"].cpu().numpy().any()
    assert float(o["E"][0]) == pytest.approx(2 * w.xi0[0]) and float(o["E"][1]) == 0.0
    assert np.array_equal(p.cpu().numpy(), two)
    pot.close()


def test_md_loop_through_the_large_system_kernels(lib, torch):
    """The MD loop on the sliced K1 / K3 (forced), where a list with a skin is compacted every step (MTP_OPT_SKIN_LIST):
    the total energy is conserved to a small fraction of the kinetic energy gained, and rebuilding every 5 steps at a
    1 A skin gives the trajectory of rebuilding every step at no skin."""
    w = make_workload(3, n_basis_of(16), cells=12)
    pot = gpu_pot(lib, w)
    pot.set_option(lib.OPT_VARIANT, lib.VARIANT_THREAD)
    pos0, types = torch.as_tensor(w.pos).cuda(), torch.as_tensor(w.types).cuda()
    mass = np.full(w.n_species, 55.845)
    cap = int(w.nnz * 1.9) + 1024
    res = {}
    for every, skin in ((1, 0.0), (5, 1.0)):
        pos, vel = pos0.clone(), torch.zeros_like(pos0)
        e0 = pot.md_run(pos, vel, types, w.box, mass, 2e-9, 0, every, skin, cap)["E"].cpu().numpy().sum()
        o = pot.md_run(pos, vel, types, w.box, mass, 2e-9, 40, every, skin, cap)
        torch.cuda.synchronize()
        E = o["E"].cpu().numpy()
        assert o["info"].cpu().tolist()[1] == 0 and o["info"].cpu().tolist()[0] <= cap
        assert pot.get_option(lib.INFO_INPUT_ERRORS) == 0 and pot.get_option(lib.INFO_SCRATCH_OVERFLOW) == 0
        assert E[1] > 0 and abs(E.sum() - e0) < 1e-4 * E[1]
        res[every] = pos.cpu().numpy()
    d = res[1] - res[5]
    L = w.box[0, 0]
    d -= np.round(d / L) * L
    assert np.abs(d).max() < 1e-10
    pot.close()
