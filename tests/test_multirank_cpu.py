"""World-size-2 gloo test (CPU) of bench.py's N > 1 host logic: replicas only, so
the only cross-rank step is the max-over-ranks timing and the whole-job rate built from it."""
import os
import socket
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    dev = torch.device("cpu")
    local_s = 0.010 * (rank + 1)                      # rank 1 is the slow one
    t = bench.max_over_ranks(local_s, dist, dev)
    v = bench.whole_job_rate(1000, 5, local_s, world, dist, dev)
    dist.barrier()
    out.put((rank, t, v))
    dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_rate():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, t, v in res:
        assert t == pytest.approx(0.020)              # both ranks see the slowest rank's time
        assert v == pytest.approx(2 * 1000 * 5 / 0.020)


def test_single_process_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(1.5, None, None) == 1.5
    assert bench.whole_job_rate(10, 2, 0.5, 1, None, None) == 40.0


# ---------------------------------------------------------------- sharded evaluation
def _oracle_rows(w, pot, lo, hi, off_w, idx_w, shift_w):
    """One rank's partial sums from the oracle, computed from the WINDOW's list only (offsets from 0, global indices)."""
    import numpy as np
    from oracle import mtp as omtp
    n = w.n_atoms
    off = np.zeros(n + 1, dtype=np.int64)                 # rows outside the window are empty
    off[lo:hi + 1] = off_w
    off[hi + 1:] = off_w[-1]
    o = omtp.evaluate(pot, w.pos, w.types, w.box, off, idx_w, shift_w, atoms=range(lo, hi))
    return o


def _shard_worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    import numpy as np
    from oracle import mtp as omtp
    from workloads import make_workload
    from _util import n_basis_of, oracle_pot
    from paper_2510_00193_b200 import sharded
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = make_workload(0, n_basis_of(10), with_ainv=True)
    pot = oracle_pot(w)
    lo, hi = sharded.balanced_row_range(w.off, rank, world)
    off_w, idx_w, shift_w = sharded.window_list(w.off, w.idx, w.shift, lo, hi)
    part = {}

    def compute_rows(a, b):
        o = _oracle_rows(w, pot, a, b, off_w, idx_w, shift_w)
        part["B"] = o["B"]
        return dict(E=torch.tensor([o["E"]]), Ei=torch.from_numpy(o["E_i"].copy()), F=torch.from_numpy(o["F"].copy()),
                    virial=torch.from_numpy(omtp.virial6(o["W"])))

    res = sharded.sharded_compute(compute_rows, dist, w.n_atoms, lo, hi)

    def grade_rows(a, b):
        g = np.zeros(w.n_atoms)
        g[a:b] = omtp.grade_neighbourhood(part["B"][a:b], w.Ainv)
        return dict(gamma_atom=torch.from_numpy(g), Bsum=torch.from_numpy(part["B"][a:b].sum(axis=0)))

    gr = sharded.sharded_grade(grade_rows, lambda s: omtp.grade_configuration(s.numpy()[None, :], w.Ainv)[0], dist, lo, hi)
    dist.barrier()
    out.put((rank, lo, hi, float(res["E"][0]), res["Ei"].numpy(), res["F"].numpy(), res["virial"].numpy(),
             gr["gamma_atom"].numpy(), float(gr["gamma_cfg"])))
    dist.destroy_process_group()


def test_sharded_evaluation_world_size_2_equals_the_whole():
    """Two ranks, contiguous atom ranges balanced by pair count, each evaluating its window from its own CSR rows
    (here with the oracle); one all-reduce of F, E, virial, E_i, one of sum B and the grades.  Both ranks end with the
    unsharded result."""
    import numpy as np
    from oracle import mtp as omtp
    from workloads import make_workload
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from _util import n_basis_of, oracle_pot
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_shard_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted((q.get(timeout=120) for _ in range(world)), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    w = make_workload(0, n_basis_of(10), with_ainv=True)
    full = omtp.evaluate(oracle_pot(w), w.pos, w.types, w.box, w.off, w.idx, w.shift)
    g_atom = omtp.grade_neighbourhood(full["B"], w.Ainv)
    g_cfg = omtp.grade_configuration(full["B"], w.Ainv)[0]
    assert res[0][1] == 0 and res[0][2] == res[1][1] and res[1][2] == w.n_atoms and 0 < res[0][2] < w.n_atoms
    fs = np.abs(full["F"]).max()
    for rank, lo, hi, E, Ei, F, vir, ga, gc in res:
        assert E == pytest.approx(full["E"], rel=1e-13)
        assert np.array_equal(Ei, full["E_i"])                       # every E_i is computed by exactly one rank
        assert np.abs(F - full["F"]).max() <= 1e-12 * fs             # partial sums added in another order
        assert np.abs(vir - omtp.virial6(full["W"])).max() <= 1e-12 * np.abs(full["W"]).max()
        assert np.array_equal(ga, g_atom) and gc == pytest.approx(g_cfg, rel=1e-12)


def test_row_ranges_cover_the_atoms_once():
    sys.path.insert(0, ROOT)
    import numpy as np
    from paper_2510_00193_b200 import sharded
    for n, world in ((10, 3), (128, 8), (5, 8), (0, 2)):
        r = [sharded.row_range(n, k, world) for k in range(world)]
        assert r[0][0] == 0 and r[-1][1] == n and all(r[k][1] == r[k + 1][0] for k in range(world - 1))
        assert max(b - a for a, b in r) - min(b - a for a, b in r) <= 1
    off = np.concatenate([[0], np.cumsum([50] * 10 + [5] * 100)])
    r = [sharded.balanced_row_range(off, k, 4) for k in range(4)]
    assert r[0][0] == 0 and r[-1][1] == 110 and all(r[k][1] == r[k + 1][0] for k in range(3))
    pairs = [off[b] - off[a] for a, b in r]
    assert max(pairs) - min(pairs) <= 50
    o, i, s = sharded.window_list(off, np.arange(off[-1], dtype=np.int32), None, 3, 12)
    assert o[0] == 0 and o[-1] == off[12] - off[3] and i[0] == off[3] and s is None
