"""-m gpu: one rank's share of a sharded evaluation (mtp_compute_rows / mtp_grade_rows / mtp_grade_cfg_from_sum; SURVEY.md
8(e), 8(f)-3).  One GPU stands in for the ranks by evaluating the windows one after the other (no kernel waits on
another); their partial sums, added on the host as the all-reduce would, are compared with the oracle and with the
unsharded call.  The collectives themselves run over gloo in tests/test_multirank_cpu.py."""
import numpy as np
import pytest

from oracle import mtp as omtp
from workloads import make_workload
from paper_2510_00193_b200 import sharded
from _util import n_basis_of, gpu_pot, oracle_pot, to_dev, scales

pytestmark = pytest.mark.gpu
TOL_E, TOL_F = 1e-10, 1e-9


@pytest.fixture(scope="module")
def torch():
    import torch as t
    assert t.cuda.is_available()
    return t


@pytest.mark.parametrize("ci,cells,world", [(0, None, 2), (1, 5, 3), (3, 6, 4)])
def test_windows_add_up_to_the_whole(lib, torch, ci, cells, world):
    w = make_workload(ci, n_basis_of([10, 16, 20, 16][ci]), cells=cells, with_ainv=True)
    pot = gpu_pot(lib, w)
    if ci == 3:
        pot.set_option(lib.OPT_CHUNK_ATOMS, 256)                      # several chunks inside a window
    d = to_dev(w, torch)
    Ainv = torch.as_tensor(w.Ainv).cuda()
    whole = pot.compute(d["pos"], d["types"], w.box, d["off"], d["idx"], d["shift"], d["rev"])
    gwhole = pot.grade(d["pos"], d["types"], w.box, d["off"], d["idx"], Ainv, d["shift"], mode=2)
    torch.cuda.synchronize()
    E, F, vir = 0.0, np.zeros((w.n_atoms, 3)), np.zeros(6)
    Ei, ga, Bsum = np.zeros(w.n_atoms), np.zeros(w.n_atoms), torch.zeros(w.xi.shape[0], dtype=torch.float64, device="cuda")
    covered = 0
    for rank in range(world):
        lo, hi = sharded.balanced_row_range(w.off, rank, world)
        off_w, idx_w, shift_w = sharded.window_list(w.off, w.idx, w.shift, lo, hi)
        t = lambda a: torch.as_tensor(a).cuda()
        o = pot.compute_rows(d["pos"], d["types"], w.box, lo, hi, t(off_w), t(idx_w), t(shift_w))
        g = pot.grade_rows(d["pos"], d["types"], w.box, lo, hi, t(off_w), t(idx_w), Ainv, t(shift_w))
        torch.cuda.synchronize()
        ei = o["Ei"].cpu().numpy()
        assert not ei[:lo].any() and not ei[hi:].any()                 # only the window's entries are written
        E += float(o["E"][0]); F += o["F"].cpu().numpy(); vir += o["virial"].cpu().numpy(); Ei += ei
        ga += g["gamma_atom"].cpu().numpy(); Bsum += g["Bsum"]
        covered += hi - lo
    assert covered == w.n_atoms
    gcfg = float(pot.grade_cfg_from_sum(Bsum, Ainv)[0])
    assert pot.get_option(lib.INFO_INPUT_ERRORS) == 0
    # against the unsharded call: E_i and the neighbourhood grades bit for bit (same kernels on the same rows), sums to rounding
    assert np.array_equal(Ei, whole["Ei"].cpu().numpy()) and np.array_equal(ga, gwhole["gamma_atom"].cpu().numpy())
    assert gcfg == pytest.approx(float(gwhole["gamma_cfg"][0]), rel=1e-12)
    # against the oracle
    opot = oracle_pot(w)
    ref = omtp.evaluate(opot, w.pos, w.types, w.box, w.off, w.idx, w.shift)
    sE, sF = scales(opot, ref, w.off, w.idx)
    assert np.all(np.abs(Ei - ref["E_i"]) <= TOL_E * sE) and abs(E - ref["E"]) <= TOL_E * sE.sum()
    assert np.all(np.abs(F - ref["F"]) <= TOL_F * sF[:, None])
    sW = max(1.0, np.abs(ref["W"]).max()) * w.off[-1]
    assert np.all(np.abs(vir - omtp.virial6(ref["W"])) <= 1e-10 * sW)
    assert np.allclose(ga, omtp.grade_neighbourhood(ref["B"], w.Ainv), rtol=1e-9, atol=0)
    assert gcfg == pytest.approx(omtp.grade_configuration(ref["B"], w.Ainv)[0], rel=1e-9)
    pot.close()


def test_window_rules(lib, torch):
    w = make_workload(0, n_basis_of(10))
    pot = gpu_pot(lib, w)
    d = to_dev(w, torch)
    t = lambda a: torch.as_tensor(a).cuda()
    off_w, idx_w, shift_w = sharded.window_list(w.off, w.idx, w.shift, 10, 20)
    pot.set_option(lib.OPT_FORCE_MODE, lib.FORCE_GATHER)               # a window has no reverse pairs
    with pytest.raises(lib.MtpError) as e:
        pot.compute_rows(d["pos"], d["types"], w.box, 10, 20, t(off_w), t(idx_w), t(shift_w))
    assert e.value.code == lib.EINVAL
    pot.set_option(lib.OPT_FORCE_MODE, lib.FORCE_AUTO)
    with pytest.raises(lib.MtpError):
        pot.compute_rows(d["pos"], d["types"], w.box, 10, w.n_atoms + 1, t(off_w), t(idx_w), t(shift_w))
    o = pot.compute_rows(d["pos"], d["types"], w.box, 7, 7, t(np.zeros(1, dtype=np.int64)), t(np.zeros(0, dtype=np.int32)), None)
    torch.cuda.synchronize()
    assert float(o["E"][0]) == 0.0 and not o["F"].cpu().numpy().any()  # an empty window
    pot.close()
