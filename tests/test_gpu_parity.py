"""-m gpu: element-by-element parity of the CUDA path (through the C ABI) with the oracle.

Tolerances (BASELINE.json north_star, read per DESIGN.md G16 as relative to the scale of
the summed terms): |dE_i| <= 1e-10 s_E, |dF| <= 1e-9 s_F, virial rel 1e-10, grades rel 1e-9.
"""
import numpy as np
import pytest

from oracle import mtp as omtp
from workloads import make_workload, random_cluster, Workload, reverse_index
from _util import n_basis_of, oracle_pot, gpu_pot, to_dev, scales

pytestmark = pytest.mark.gpu
TOL_E, TOL_F, TOL_W, TOL_G = 1e-10, 1e-9, 1e-10, 1e-9


@pytest.fixture(scope="module")
def torch():
    import torch as t
    assert t.cuda.is_available()
    return t


def assert_specialised(lib, pot):
    """The contraction kernels that ran are the NVRTC-specialised ones (the product path), not the interpreter:
    two kernels (energy + adjoint, values) per program, and the handle reports no fallback."""
    n_prog = pot.get_option(lib.INFO_TREE_PROGRAMS)
    assert n_prog >= 1 and pot.get_option(lib.INFO_TREE_KERNELS) == 2 * n_prog, pot.last_error()
    assert pot.get_option(lib.OPT_TREE_CODEGEN) == 1
    return n_prog


def run_gpu(lib, torch, w, pot=None, opts=None, interp=False):
    """One mtp_compute through the C ABI.  interp: the table interpreter instead of the specialised kernels."""
    pot = gpu_pot(lib, w) if pot is None else pot
    for k, v in (opts or {}).items():
        pot.set_option(k, v)
    if interp:
        pot.set_option(lib.OPT_TREE_CODEGEN, 0)
        assert pot.get_option(lib.OPT_TREE_CODEGEN) == 0
    else:
        assert_specialised(lib, pot)
    d = to_dev(w, torch)
    out = pot.compute(d["pos"], d["types"], w.box, d["off"], d["idx"], d["shift"], d["rev"])
    torch.cuda.synchronize()
    return {k: v.cpu().numpy() for k, v in out.items()}, pot, d


def check(w, ref, got, opot):
    sE, sF = scales(opot, ref, w.off, w.idx)
    assert np.all(np.abs(got["Ei"] - ref["E_i"]) <= TOL_E * sE), np.abs((got["Ei"] - ref["E_i"]) / sE).max()
    assert abs(got["E"][0] - ref["E"]) <= TOL_E * sE.sum()
    assert np.all(np.abs(got["F"] - ref["F"]) <= TOL_F * sF[:, None]), np.abs((got["F"] - ref["F"]) / sF[:, None]).max()
    # virial: relative to the sum of |r_a d_b| magnitudes
    rv = np.concatenate([omtp.pair_vectors(i, w.pos, w.box, w.off, w.idx, w.shift)[1] for i in range(w.n_atoms)])
    sW = max(1.0, np.abs(rv[:, :, None] * ref["d"][:, None, :]).sum())
    assert np.all(np.abs(got["virial"] - omtp.virial6(ref["W"])) <= TOL_W * sW)


CASES = [(0, None), (1, 5), (2, 4), (3, 3)]


@pytest.mark.parametrize("ci,cells", CASES)
def test_energy_force_virial_parity(lib, torch, ci, cells):
    w = make_workload(ci, n_basis_of([10, 16, 20, 16][ci]), cells=cells)
    opot = oracle_pot(w)
    ref = omtp.evaluate(opot, w.pos, w.types, w.box, w.off, w.idx, w.shift)
    for variant in (lib.VARIANT_THREAD, lib.VARIANT_BLOCK):
        for mode in (lib.FORCE_GATHER, lib.FORCE_ATOMIC):
            got, pot, _ = run_gpu(lib, torch, w, opts={lib.OPT_VARIANT: variant, lib.OPT_FORCE_MODE: mode})
            check(w, ref, got, opot)
            pot.close()
    got, pot, _ = run_gpu(lib, torch, w, interp=True)          # the fallback form of K2 against the oracle as well
    check(w, ref, got, opot)
    pot.close()


def test_config1_meets_the_absolute_tolerances_as_written(lib, torch):
    """BASELINE.json configs[0] (128 atoms, level 10) at full size against north_star's numbers read literally:
    |dE_i| <= 1e-10 eV, |dF| <= 1e-9 eV/A, virial relative 1e-10 (at level 10 the magnitudes
    still allow it)."""
    w = make_workload(0, n_basis_of(10))
    assert w.n_atoms == 128
    opot = oracle_pot(w)
    ref = omtp.evaluate(opot, w.pos, w.types, w.box, w.off, w.idx, w.shift)
    got, pot, _ = run_gpu(lib, torch, w)
    pot.close()
    assert np.abs(got["Ei"] - ref["E_i"]).max() <= 1e-10
    assert np.abs(got["F"] - ref["F"]).max() <= 1e-9
    W6 = omtp.virial6(ref["W"])
    assert np.abs(got["virial"] - W6).max() <= 1e-10 * np.abs(W6).max()


def test_config2_full_size_energy_force_virial(lib, torch):
    """BASELINE.json configs[1] at its stated size (2 000 atoms, level 16): every E_i, F_k and the virial."""
    w = make_workload(1, n_basis_of(16))
    assert w.n_atoms == 2000
    opot = oracle_pot(w)
    ref = omtp.evaluate(opot, w.pos, w.types, w.box, w.off, w.idx, w.shift)
    got, pot, _ = run_gpu(lib, torch, w)
    check(w, ref, got, opot)
    pot.close()


def sheared_workload(lev, n_mu, seed, n, S):
    """Triclinic periodic box (rows = lattice vectors, all heights > 2 R_cut) with random atoms."""
    rng = np.random.default_rng(seed)
    box = np.array([[12.5, 0.0, 0.0], [3.1, 12.0, 0.0], [-2.2, 1.7, 11.6]])
    pos = rng.uniform(0, 1, (n, 3)) @ box
    types = rng.integers(0, S, n).astype(np.int32)
    off, idx, sh = omtp.brute_force_neighbours(pos, box, 5.0)
    nb = n_basis_of(lev)
    return Workload(name="sheared", lev_max=lev, n_mu=n_mu, n_beta=8, r_min=2.0, r_cut=5.0, n_species=S,
                    box=box, pos=pos, types=types, c=rng.uniform(-0.1, 0.1, (S, S, n_mu, 8)),
                    xi0=rng.uniform(-0.1, 0.1, S), xi=rng.uniform(-0.1, 0.1, nb), off=off, idx=idx,
                    shift=sh, rev=reverse_index(off, idx, sh))


@pytest.mark.parametrize("lev,n_mu", [(10, 3), (16, 4)])
def test_triclinic_box_with_shifts_and_with_minimum_image(lib, torch, lev, n_mu):
    """A sheared box reaches the CUDA path: the image-shift table s.H and the inverse-box columns of the minimum
    image (csrc/api.cu box_setup, csrc/pair_kernels.cuh pair_vector) against the oracle, both ways."""
    w = sheared_workload(lev, n_mu, 41, 30, 2)
    assert np.abs(w.shift).max() == 1
    opot = oracle_pot(w)
    ref = omtp.evaluate(opot, w.pos, w.types, w.box, w.off, w.idx, w.shift)
    got, pot, d = run_gpu(lib, torch, w)
    check(w, ref, got, opot)
    out = pot.compute(d["pos"], d["types"], w.box, d["off"], d["idx"], None, d["rev"])       # minimum image
    torch.cuda.synchronize()
    check(w, ref, {k: v.cpu().numpy() for k, v in out.items()}, opot)
    pot.close()


def test_rejected_neighbour_entries_are_counted(lib, torch):
    """include/mtp_b200.h: image shifts outside {-1,0,1}^3 (and indices outside [0, N)) do not fit the packed
    neighbour word; they are dropped and reported through MTP_INFO_INPUT_ERRORS instead of aliasing silently."""
    w = make_workload(0, n_basis_of(10))
    pot = gpu_pot(lib, w)
    d = to_dev(w, torch)
    assert pot.get_option(lib.INFO_INPUT_ERRORS) == 0
    pot.compute(d["pos"], d["types"], w.box, d["off"], d["idx"], d["shift"], d["rev"])
    assert pot.get_option(lib.INFO_INPUT_ERRORS) == 0
    bad = d["shift"].clone()
    bad[5, 0] = 2
    bad[77, 2] = -3
    pot.compute(d["pos"], d["types"], w.box, d["off"], d["idx"], bad, d["rev"])
    assert pot.get_option(lib.INFO_INPUT_ERRORS) == 2
    assert pot.get_option(lib.INFO_INPUT_ERRORS) == 0          # reading resets the counter
    pot.close()


def test_per_pair_scratch_is_bounded_by_the_chunk(lib, torch):
    """a10 (north_star 'a chunk scheduler that bounds per-pair scratch'): with the paper's example
    chunk of 32 768 atoms the workspace of config 4 (1 048 576 atoms, 47.2 M pairs) stays below 200 MB in the
    deterministic force mode (d_ij for all pairs would be 1.5 GB); a chunk with more pairs than the scratch was sized
    for is reported, not silently wrong."""
    w = make_workload(1, n_basis_of(16), cells=5)
    pot = gpu_pot(lib, w)
    pot.set_option(lib.OPT_FORCE_MODE, lib.FORCE_GATHER)
    pot.set_option(lib.OPT_CHUNK_ATOMS, 32768)
    assert pot.workspace_bytes(1048576, 47194874) < 200e6
    pot.set_option(lib.OPT_CHUNK_ATOMS, 262144)
    assert pot.workspace_bytes(1048576, 47194874) < 1.3e9        # four chunks: a quarter of the pairs
    pot.set_option(lib.OPT_CHUNK_ATOMS, 0)
    assert pot.workspace_bytes(1048576, 47194874) < 4.2e9        # automatic: one chunk within the 4 GB budget for M + G
    d = to_dev(w, torch)
    pot.set_option(lib.OPT_CHUNK_ATOMS, 64)
    pot.set_option(lib.OPT_CHUNK_PAIRS, 100)                      # far too small for 64 atoms x ~54 neighbours
    pot.compute(d["pos"], d["types"], w.box, d["off"], d["idx"], d["shift"], d["rev"])
    assert pot.get_option(lib.INFO_SCRATCH_OVERFLOW) > 0
    pot.close()


def test_chunked_equals_unchunked_and_gather_is_deterministic(lib, torch):
    w = make_workload(1, n_basis_of(16), cells=5)
    a, pot, d = run_gpu(lib, torch, w, opts={lib.OPT_FORCE_MODE: lib.FORCE_GATHER})
    b, _, _ = run_gpu(lib, torch, w, pot=pot)
    assert np.array_equal(a["F"], b["F"]) and np.array_equal(a["Ei"], b["Ei"]) and np.array_equal(a["virial"], b["virial"])
    c, _, _ = run_gpu(lib, torch, w, pot=pot, opts={lib.OPT_CHUNK_ATOMS: 77})   # ragged last chunk
    assert np.array_equal(a["Ei"], c["Ei"])
    # forces are assembled chunk by chunk in stream order (per-pair scratch exists for one chunk at a time): same
    # per-pair values, another summation order -> equal to rounding, and bit-identical from run to run
    assert np.allclose(a["F"], c["F"], rtol=0, atol=1e-13 * np.abs(a["F"]).max())
    assert np.allclose(a["virial"], c["virial"], rtol=1e-12)
    c2, _, _ = run_gpu(lib, torch, w, pot=pot)
    assert np.array_equal(c["F"], c2["F"]) and np.array_equal(c["virial"], c2["virial"])
    assert pot.get_option(lib.INFO_SCRATCH_OVERFLOW) == 0 and pot.get_option(lib.INFO_INPUT_ERRORS) == 0
    pot.set_option(lib.OPT_CHUNK_ATOMS, 0)
    # minimum image instead of explicit shifts gives the same pairs here (box > 2 R_cut)
    out = pot.compute(d["pos"], d["types"], w.box, d["off"], d["idx"], None, d["rev"])
    torch.cuda.synchronize()
    assert np.allclose(out["F"].cpu().numpy(), a["F"], rtol=0, atol=1e-9 * np.abs(a["F"]).max())
    pot.close()


def cluster_workload(lev, n_mu, seed, n, S, box_len=11.0, r_list=5.0, n_beta=8):
    pos, types, box = random_cluster(seed, n, box_len, n_species=S)
    off, idx, sh = omtp.brute_force_neighbours(pos, box, r_list)
    rng = np.random.default_rng(seed + 1)
    nb = n_basis_of(lev)
    return Workload(name="cluster", lev_max=lev, n_mu=n_mu, n_beta=n_beta, r_min=2.0, r_cut=5.0, n_species=S,
                    box=box, pos=pos, types=types, c=rng.uniform(-0.1, 0.1, (S, S, n_mu, n_beta)),
                    xi0=rng.uniform(-0.1, 0.1, S), xi=rng.uniform(-0.1, 0.1, nb), off=off, idx=idx,
                    shift=sh, rev=reverse_index(off, idx, sh))


@pytest.mark.parametrize("lev,n_mu,n", [(10, 3, 40), (16, 4, 30), (24, 6, 14)])
def test_ragged_cluster_with_skin_and_short_pairs(lib, torch, lev, n_mu, n):
    """Random cluster: ragged rows, pairs below R_min (G2), list with a skin (G3)."""
    w = cluster_workload(lev, n_mu, 21, n, 2, r_list=5.5)
    opot = oracle_pot(w)
    ref = omtp.evaluate(opot, w.pos, w.types, w.box, w.off, w.idx, w.shift)
    got, pot, _ = run_gpu(lib, torch, w)
    if lev >= 20:
        assert pot.get_option(lib.INFO_TREE_PROGRAMS) > 1          # partitioned: top program + group programs
    check(w, ref, got, opot)
    pot.close()
    got, pot, _ = run_gpu(lib, torch, w, interp=True)
    check(w, ref, got, opot)
    pot.close()


@pytest.mark.parametrize("n_beta", [1, 2, 5, 12])
def test_radial_basis_sizes_other_than_eight(lib, torch, n_beta):
    """The BASELINE configurations all have 8 Chebyshev polynomials (a compile-time size in K1 / K3); any other size
    takes the run-time loop.  Small-system kernels, then the large-system (sliced) kernels forced on the same cluster."""
    w = cluster_workload(16, 4, 33, 36, 3, r_list=5.3, n_beta=n_beta)
    opot = oracle_pot(w)
    ref = omtp.evaluate(opot, w.pos, w.types, w.box, w.off, w.idx, w.shift)
    for variant in (lib.VARIANT_AUTO, lib.VARIANT_THREAD):
        for mode in (lib.FORCE_GATHER, lib.FORCE_ATOMIC):
            got, pot, _ = run_gpu(lib, torch, w, opts={lib.OPT_VARIANT: variant, lib.OPT_FORCE_MODE: mode})
            check(w, ref, got, opot)
            pot.close()


@pytest.mark.parametrize("S", [5, 8])
def test_many_species(lib, torch, S):
    """More species than any BASELINE configuration: S^2 coefficient blocks staged in shared memory (c[z_i][z_j] is not
    symmetric: reading G6), small- and large-system kernels."""
    w = cluster_workload(10, 3, 44 + S, 48, S, r_list=5.0)
    assert len(set(w.types.tolist())) == S
    opot = oracle_pot(w)
    ref = omtp.evaluate(opot, w.pos, w.types, w.box, w.off, w.idx, w.shift)
    for variant in (lib.VARIANT_AUTO, lib.VARIANT_THREAD):
        got, pot, _ = run_gpu(lib, torch, w, opts={lib.OPT_VARIANT: variant})
        check(w, ref, got, opot)
        pot.close()


def test_level24_lattice_sample_and_grades(lib, torch):
    """Config-5 shape at reduced size: B, E_i on sampled atoms; both grade modes."""
    nb = n_basis_of(24)
    w = make_workload(4, nb, cells=4, with_ainv=True)
    opot = oracle_pot(w)
    sample = list(range(0, w.n_atoms, 9))
    ref = omtp.evaluate(opot, w.pos, w.types, w.box, w.off, w.idx, w.shift, atoms=sample, want_grad=False)
    pot = gpu_pot(lib, w)
    d = to_dev(w, torch)
    Ainv = torch.as_tensor(w.Ainv).cuda()
    g = pot.grade(d["pos"], d["types"], w.box, d["off"], d["idx"], Ainv, d["shift"], mode=2, want_B=True)
    torch.cuda.synchronize()
    B = g["B"].cpu().numpy()
    sB = np.maximum(1.0, np.abs(ref["B"][sample]).max(axis=1))[:, None]
    assert np.all(np.abs(B[sample] - ref["B"][sample]) <= 1e-10 * np.maximum(np.abs(ref["B"][sample]), 1e-6 * sB))
    # grades from the oracle on the GPU's own B would hide B errors: use the oracle's B rows
    ga = g["gamma_atom"].cpu().numpy()
    want = omtp.grade_neighbourhood(ref["B"][sample], w.Ainv)
    assert np.allclose(ga[sample], want, rtol=TOL_G)
    # configuration mode: needs every atom's B; check the kernel against the oracle formula on the
    # GPU-produced (and above validated-by-sample) B matrix, and Bsum against a plain column sum
    gc, Bsum = omtp.grade_configuration(B, w.Ainv)
    assert np.allclose(g["Bsum"].cpu().numpy(), Bsum, rtol=1e-12)
    assert g["gamma_cfg"].cpu().numpy()[0] == pytest.approx(gc, rel=TOL_G)
    pot.close()


def test_grades_full_parity_small(lib, torch):
    w = make_workload(1, n_basis_of(16), cells=4, with_ainv=True)
    opot = oracle_pot(w)
    ref = omtp.evaluate(opot, w.pos, w.types, w.box, w.off, w.idx, w.shift, want_grad=False)
    pot = gpu_pot(lib, w)
    d = to_dev(w, torch)
    for chunk in (0, 50):
        pot.set_option(lib.OPT_CHUNK_ATOMS, chunk)
        g = pot.grade(d["pos"], d["types"], w.box, d["off"], d["idx"], torch.as_tensor(w.Ainv).cuda(), d["shift"])
        torch.cuda.synchronize()
        assert np.allclose(g["gamma_atom"].cpu().numpy(), omtp.grade_neighbourhood(ref["B"], w.Ainv), rtol=TOL_G)
        gc, Bsum = omtp.grade_configuration(ref["B"], w.Ainv)
        assert np.allclose(g["Bsum"].cpu().numpy(), Bsum, rtol=1e-10, atol=1e-10 * np.abs(ref["B"]).sum(axis=0).max())
        assert g["gamma_cfg"].cpu().numpy()[0] == pytest.approx(gc, rel=TOL_G)
    pot.close()


def test_edge_cases(lib, torch):
    import torch as t
    w = make_workload(0, n_basis_of(10))
    pot = gpu_pot(lib, w)
    dev = t.device("cuda:0")
    # N = 0
    z = lambda dt, *s: t.zeros(*s, dtype=dt, device=dev)
    out = pot.compute(z(t.float64, 0, 3), z(t.int32, 0), w.box, z(t.int64, 1), z(t.int32, 0))
    t.cuda.synchronize()
    assert out["E"].item() == 0.0 and np.all(out["virial"].cpu().numpy() == 0.0)
    # isolated atoms: E_i = xi0, F = 0 (G20)
    pos = t.tensor([[1.0, 1.0, 1.0], [20.0, 20.0, 20.0]], dtype=t.float64, device=dev)
    out = pot.compute(pos, z(t.int32, 2), np.eye(3) * 40, z(t.int64, 3), z(t.int32, 0))
    t.cuda.synchronize()
    assert np.array_equal(out["Ei"].cpu().numpy(), np.full(2, w.xi0[0])) and np.all(out["F"].cpu().numpy() == 0)
    # error codes: box too small for minimum image, workspace too small
    d = to_dev(w, t)
    with pytest.raises(lib.MtpError) as e:
        pot.compute(d["pos"], d["types"], np.eye(3) * 9.0, d["off"], d["idx"], None, d["rev"])
    assert e.value.code == lib.EBOX
    pot.close()


def test_host_path_matches_device_path(lib, torch):
    w = make_workload(1, n_basis_of(16), cells=4)
    got, pot, _ = run_gpu(lib, torch, w)
    h = pot.compute_host(w.pos, w.types, w.box, w.off, w.idx, w.shift, w.rev)
    assert np.array_equal(h["F"], got["F"]) and np.array_equal(h["Ei"], got["Ei"]) and h["E"][0] == got["E"][0]
    pot.close()


def test_cuda_graph_replay_of_a_call_is_bit_identical(lib, torch):
    """mtp_compute only enqueues on the caller's stream (include/mtp_b200.h): a captured call replays exactly."""
    w = make_workload(1, n_basis_of(16), cells=4)
    a, pot, d = run_gpu(lib, torch, w, opts={lib.OPT_FORCE_MODE: lib.FORCE_GATHER})
    out = pot.compute(d["pos"], d["types"], w.box, d["off"], d["idx"], d["shift"], d["rev"])
    torch.cuda.synchronize()
    side = torch.cuda.Stream()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=side):
        pot.compute(d["pos"], d["types"], w.box, d["off"], d["idx"], d["shift"], d["rev"], out=out)
    for v in out.values():
        v.fill_(float("nan"))
    g.replay()
    torch.cuda.synchronize()
    for k in ("E", "Ei", "F", "virial"):
        assert np.array_equal(out[k].cpu().numpy(), a[k]), k
    d["pos"].add_(0.01 * torch.randn_like(d["pos"]))      # same buffers, new coordinates: the graph follows the data
    g.replay()
    torch.cuda.synchronize()
    b = {k: v.cpu().numpy().copy() for k, v in out.items()}
    ref = pot.compute(d["pos"], d["types"], w.box, d["off"], d["idx"], d["shift"], d["rev"])
    torch.cuda.synchronize()
    for k in ("E", "Ei", "F", "virial"):
        assert np.array_equal(ref[k].cpu().numpy(), b[k]), k
    pot.close()


def test_graph_behind_the_abi_is_bit_identical_and_follows_the_data(lib, torch):
    """mtp_graph_capture / mtp_graph_launch: the small-system path (one launch per evaluation).  Capture runs nothing;
    a launch equals mtp_compute bit for bit, also after the coordinates changed in place, on any stream."""
    for ci, cells in ((0, None), (1, 4)):
        w = make_workload(ci, n_basis_of([10, 16][ci]), cells=cells)
        a, pot, d = run_gpu(lib, torch, w, opts={lib.OPT_FORCE_MODE: lib.FORCE_GATHER})
        pot.set_option(lib.OPT_PROFILE, 1)                             # capture has to switch the timing events off itself
        n0 = lib.launch_count()
        g, out = pot.graph(d["pos"], d["types"], w.box, d["off"], d["idx"], d["shift"], d["rev"])
        assert pot.get_option(lib.OPT_PROFILE) == 1
        for v in out.values():
            v.fill_(float("nan"))
        torch.cuda.synchronize()
        assert np.isnan(out["F"].cpu().numpy()).all()                  # nothing ran at capture
        g.launch()
        torch.cuda.synchronize()
        for k in ("E", "Ei", "F", "virial"):
            assert np.array_equal(out[k].cpu().numpy(), a[k]), k
        d["pos"].add_(0.01 * torch.randn_like(d["pos"]))
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        g.launch(stream=side)
        g.launch(stream=side)
        side.synchronize()
        ref = pot.compute(d["pos"], d["types"], w.box, d["off"], d["idx"], d["shift"], d["rev"])
        torch.cuda.synchronize()
        for k in ("E", "Ei", "F", "virial"):
            assert np.array_equal(ref[k].cpu().numpy(), out[k].cpu().numpy()), k
        g.close()
        pot.close()


def test_unaligned_list_arrays_take_the_scalar_loads(lib, torch):
    """The pair packer reads indices 16 bytes and shifts 4 bytes at a time when the arrays are aligned; list arrays that
    start at an odd element (a view into a larger buffer) go through the scalar loads: same result bit for bit."""
    w = make_workload(1, n_basis_of(16), cells=4)
    a, pot, d = run_gpu(lib, torch, w, opts={lib.OPT_FORCE_MODE: lib.FORCE_GATHER, lib.OPT_CHUNK_ATOMS: 40})
    idx = torch.empty(w.nnz + 3, dtype=torch.int32, device="cuda")[3:]
    shift = torch.empty((w.nnz * 3 + 1,), dtype=torch.int8, device="cuda")[1:].view(w.nnz, 3)
    assert idx.data_ptr() % 16 != 0 and shift.data_ptr() % 4 != 0
    idx.copy_(d["idx"]); shift.copy_(d["shift"])
    b = pot.compute(d["pos"], d["types"], w.box, d["off"], idx, shift, d["rev"])
    torch.cuda.synchronize()
    for k in ("E", "Ei", "F", "virial"):
        assert np.array_equal(b[k].cpu().numpy(), a[k]), k
    assert pot.get_option(lib.INFO_INPUT_ERRORS) == 0
    pot.close()


def test_specialised_and_interpreted_tree_kernels_agree(lib, torch):
    """MTP_OPT_TREE_CODEGEN: the two forms of K2 sum in different orders, so they agree to rounding (relative to the
    magnitude of the summed terms), not bit for bit; each is compared with the oracle elsewhere."""
    w = make_workload(3, n_basis_of(16), cells=18)            # 23 328 atoms, 3 species, level 16
    a, pot, d = run_gpu(lib, torch, w, opts={lib.OPT_VARIANT: lib.VARIANT_THREAD}, interp=True)
    pot.close()
    b, pot, _ = run_gpu(lib, torch, w, opts={lib.OPT_VARIANT: lib.VARIANT_THREAD})
    pot.close()
    sE = np.maximum(1.0, np.abs(a["Ei"]))
    assert np.all(np.abs(a["Ei"] - b["Ei"]) <= 1e-12 * sE.max())
    assert np.all(np.abs(a["F"] - b["F"]) <= 1e-11 * np.abs(a["F"]).max())
    assert np.allclose(a["virial"], b["virial"], rtol=0, atol=1e-11 * np.abs(a["virial"]).max())


def test_large_launch_configuration_on_sampled_atoms(lib, torch):
    """The launch configuration bench.py times (config 4 structure, thread-parallel pair kernels, 64-atom
    tree CTAs, specialised K2, several chunks): E_i, F_k on sampled atoms against the oracle, sum F = 0."""
    w = make_workload(3, n_basis_of(16), cells=22)            # 42 592 atoms, 3 species, level 16
    got, pot, _ = run_gpu(lib, torch, w, opts={lib.OPT_CHUNK_ATOMS: 16384})
    assert pot.get_option(lib.OPT_VARIANT) == lib.VARIANT_AUTO
    pot.close()
    opot = oracle_pot(w)
    rng = np.random.default_rng(5)
    sample = [int(x) for x in rng.choice(w.n_atoms, 5, replace=False)]
    need = set(sample)
    for k in sample:
        need.update(int(j) for j in w.idx[w.off[k]:w.off[k + 1]])
    ref = omtp.evaluate(opot, w.pos, w.types, w.box, w.off, w.idx, w.shift, atoms=sorted(need))
    d = ref["d"]
    for k in sample:
        sE = max(1.0, np.abs(ref["B"][k] * w.xi).sum())
        assert abs(got["Ei"][k] - ref["E_i"][k]) <= TOL_E * sE
        rows = np.arange(w.off[k], w.off[k + 1])
        Fk = d[rows].sum(axis=0) - d[w.rev[rows]].sum(axis=0)
        sF = max(1.0, np.abs(d[rows]).sum() + np.abs(d[w.rev[rows]]).sum())
        assert np.all(np.abs(got["F"][k] - Fk) <= TOL_F * sF)
    assert np.all(np.abs(got["F"].sum(axis=0)) <= 1e-9 * np.abs(got["F"]).sum())


def _check_sampled(w, got, n_sample, seed):
    """E_i and F_k of sampled atoms against the oracle (the oracle evaluates the sampled atoms and their neighbours)."""
    opot = oracle_pot(w)
    rng = np.random.default_rng(seed)
    sample = [int(x) for x in rng.choice(w.n_atoms, n_sample, replace=False)]
    need = set(sample)
    for k in sample:
        need.update(int(j) for j in w.idx[w.off[k]:w.off[k + 1]])
    ref = omtp.evaluate(opot, w.pos, w.types, w.box, w.off, w.idx, w.shift, atoms=sorted(need))
    d = ref["d"]
    for k in sample:
        sE = max(1.0, np.abs(ref["B"][k] * w.xi).sum())
        assert abs(got["Ei"][k] - ref["E_i"][k]) <= TOL_E * sE
        rows = np.arange(w.off[k], w.off[k + 1])
        Fk = d[rows].sum(axis=0) - d[w.rev[rows]].sum(axis=0)
        sF = max(1.0, np.abs(d[rows]).sum() + np.abs(d[w.rev[rows]]).sum())
        assert np.all(np.abs(got["F"][k] - Fk) <= TOL_F * sF)
    assert np.all(np.abs(got["F"].sum(axis=0)) <= 1e-9 * np.abs(got["F"]).sum())


def test_full_size_config4_sampled(lib, torch):
    """BASELINE.json configs[3] at full size (1,048,576 atoms, level 16), default options = what bench.py times."""
    w = make_workload(3, n_basis_of(16))
    got, pot, _ = run_gpu(lib, torch, w)
    pot.close()
    assert w.n_atoms == 1048576
    _check_sampled(w, got, 4, 11)


def test_full_size_config3_sampled(lib, torch):
    """BASELINE.json configs[2] at full size (54,000 atoms, 2 species, level 20)."""
    w = make_workload(2, n_basis_of(20))
    got, pot, _ = run_gpu(lib, torch, w)
    assert assert_specialised(lib, pot) == lib.Table(20).plan()["groups"] + 1
    pot.close()
    assert w.n_atoms == 54000
    _check_sampled(w, got, 2, 12)


def test_full_size_config5_sampled_energy_and_grades(lib, torch):
    """BASELINE.json configs[4] at full size (250,000 atoms, level 24): E_i, B and both grade modes on sampled atoms."""
    nb = n_basis_of(24)
    w = make_workload(4, nb)
    assert w.n_atoms == 250000 and w.Ainv is not None
    opot = oracle_pot(w)
    sample = [3, 124999, 249998]
    ref = omtp.evaluate(opot, w.pos, w.types, w.box, w.off, w.idx, w.shift, atoms=sample, want_grad=False)
    pot = gpu_pot(lib, w)
    d = to_dev(w, torch)
    out = pot.compute(d["pos"], d["types"], w.box, d["off"], d["idx"], d["shift"], d["rev"])
    Ainv = torch.as_tensor(w.Ainv).cuda()
    g = pot.grade(d["pos"], d["types"], w.box, d["off"], d["idx"], Ainv, d["shift"], mode=2)
    torch.cuda.synchronize()
    Ei = out["Ei"].cpu().numpy()
    ga = g["gamma_atom"].cpu().numpy()
    want = omtp.grade_neighbourhood(ref["B"][sample], w.Ainv)
    for q, k in enumerate(sample):
        sE = max(1.0, np.abs(ref["B"][k] * w.xi).sum())
        assert abs(Ei[k] - ref["E_i"][k]) <= TOL_E * sE
        assert ga[k] == pytest.approx(want[q], rel=TOL_G)
    n_prog = assert_specialised(lib, pot)
    assert n_prog == lib.Table(24).plan()["groups"] + 1        # top program + every group program, all specialised
    # forces through the partitioned, specialised K2 (group programs seeded with dE/dS, G accumulated over the
    # groups) and K3: F_k of sampled atoms against the oracle, which evaluates them and all their neighbours
    got = {"Ei": Ei, "F": out["F"].cpu().numpy()}
    _check_sampled(w, got, 2, 13)
    # configuration mode: property that holds at any size -- gamma_cfg = max_k |Bsum . Ainv[:, k]| of the returned Bsum
    Bsum = g["Bsum"].cpu().numpy()
    assert g["gamma_cfg"].cpu().numpy()[0] == pytest.approx(np.abs(Bsum @ w.Ainv).max(), rel=TOL_G)
    pot.close()


def test_error_codes_for_bad_tables_and_small_workspace(lib, torch):
    """Errors are codes, never aborts: malformed contraction tables (MTP_EINVAL) and a short workspace (MTP_ESIZE)."""
    import ctypes as C
    from paper_2510_00193_b200 import binding as bnd
    t = lib.Table(10)
    rng = np.random.default_rng(3)
    c = rng.uniform(-0.1, 0.1, (1, 1, t.n_mu, 8))
    xi0, xi = np.zeros(1), rng.uniform(-0.1, 0.1, t.n_basis)
    bad = t.prod.copy()
    bad[0, 0] = t.n_nodes + 5                                  # source index out of range
    with pytest.raises(lib.MtpError) as e:
        lib.Potential(t, 1, 8, 2.0, 5.0, c, xi0, xi, prod=bad)
    assert e.value.code == lib.EINVAL
    bad = t.prod.copy()
    last = bad[-1].copy()                                      # a node is read before it is written
    bad[1:] = t.prod[:-1]
    bad[0] = last
    if last[0] >= t.n_basic or last[1] >= t.n_basic:
        with pytest.raises(lib.MtpError) as e:
            lib.Potential(t, 1, 8, 2.0, 5.0, c, xi0, xi, prod=bad)
        assert e.value.code == lib.EINVAL
    w = make_workload(0, t.n_basis)
    pot = gpu_pot(lib, w)
    d = to_dev(w, torch)
    n, nnz = w.n_atoms, w.nnz
    out = [torch.empty(s, dtype=torch.float64, device="cuda") for s in (1, n, (n, 3), 6)]
    ws = torch.empty(1024, dtype=torch.uint8, device="cuda")   # far too small
    boxh = (C.c_double * 9)(*[float(x) for x in np.asarray(w.box).reshape(9)])
    p = lambda x: C.c_void_p(x.data_ptr())
    rc = bnd._lib.mtp_compute(pot._h, n, p(d["pos"]), p(d["types"]), boxh, p(d["off"]), p(d["idx"]), p(d["shift"]),
                              p(d["rev"]), nnz, p(out[0]), p(out[1]), p(out[2]), p(out[3]), p(ws), ws.numel(), C.c_void_p(0))
    assert rc == lib.ESIZE
    pot.close()


def test_level28_partitioned_tree_interpreted(lib, torch):
    """Level 28 (9 739 basis functions): one atom's node values exceed shared memory, so the table only runs
    partitioned (132 group programs + top program), and with 350 000 table ops it is above the size mtp_create
    specialises: the interpreter runs, and the handle says so."""
    lev, n_mu = 28, 7
    plan = lib.Table(lev).plan()
    assert plan["partitioned"] == 1 and plan["specialised"] == 0
    w = cluster_workload(lev, n_mu, 33, 8, 2, r_list=5.0)
    opot = oracle_pot(w)
    ref = omtp.evaluate(opot, w.pos, w.types, w.box, w.off, w.idx, w.shift)
    got, pot, _ = run_gpu(lib, torch, w, interp=True)
    assert pot.get_option(lib.INFO_TREE_KERNELS) == 0 and "too large to specialise" in pot.last_error()
    check(w, ref, got, opot)
    pot.close()
