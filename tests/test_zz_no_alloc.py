"""-m gpu, collected last: mtp_neighbors_build_static, the list build that allocates nothing (its workspace is a static
device array in the library, limit MTP_NB_STATIC_MAX_ATOMS atoms), against mtp_neighbors_build with a caller workspace.
Integer work: the two lists are compared bit for bit, on two calls in a row that share the static array."""
import numpy as np
import pytest

from workloads import make_workload

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch():
    import torch as t
    assert t.cuda.is_available()
    return t


def _static(lib, torch, pos, box, r, cap):
    """outputs pre-filled with a pattern, so a stale or unwritten entry cannot pass for a result"""
    n = pos.shape[0]
    off = torch.full((n + 1,), -7, dtype=torch.int64, device="cuda")
    idx = torch.full((cap,), -7, dtype=torch.int32, device="cuda")
    shift = torch.full((cap, 3), 5, dtype=torch.int8, device="cuda")
    rev = torch.full((cap,), -7, dtype=torch.int32, device="cuda")
    info = torch.full((2,), -7, dtype=torch.int64, device="cuda")
    lib.neighbors_build_static(pos, box, r, off, idx, shift, rev, info)
    return off, idx, shift, rev, info


def test_static_workspace_list_equals_the_workspace_path_twice(lib, torch):
    """Call 1: config 2 (2 000 atoms, cubic box).  Call 2 right behind it on the same stream: fewer atoms in a sheared
    box with another cell grid -- whatever call 1 left in the shared array must not show.  Then call 1 again."""
    w = make_workload(1, 1)
    rng = np.random.default_rng(11)
    box2 = np.array([[12.5, 0.0, 0.0], [3.1, 12.0, 0.0], [-2.2, 1.7, 11.6]])
    pos2 = rng.uniform(0, 1, (150, 3)) @ box2
    cases = [(w.pos, w.box, 5.0), (pos2, box2, 5.5), (w.pos, w.box, 5.0)]
    dev = [(torch.as_tensor(np.ascontiguousarray(p)).cuda(), b, r) for p, b, r in cases]
    want = [lib.neighbors_build(p, b, r) for p, b, r in dev]                    # existing path, its own workspace
    torch.cuda.synchronize()
    got = [_static(lib, torch, p, b, r, ref["nnz"] + 64) for (p, b, r), ref in zip(dev, want)]   # back to back, no sync between
    torch.cuda.synchronize()
    for ref, (off, idx, shift, rev, info) in zip(want, got):
        n = ref["nnz"]
        assert n > 0 and ref["errors"] == 0
        assert info.cpu().tolist() == [n, 0]
        assert torch.equal(off, ref["off"])
        assert torch.equal(idx[:n], ref["idx"][:n]) and torch.equal(shift[:n], ref["shift"][:n]) and torch.equal(rev[:n], ref["rev"][:n])
        assert bool((idx[n:] == -7).all()) and bool((rev[n:] == -7).all())        # nothing written past the list


def test_static_workspace_limit_and_bad_arguments(lib, torch):
    n = lib.NB_STATIC_MAX_ATOMS + 1
    pos = torch.zeros((n, 3), dtype=torch.float64, device="cuda")
    off = torch.zeros(n + 1, dtype=torch.int64, device="cuda")
    idx = torch.zeros(8, dtype=torch.int32, device="cuda")
    shift = torch.zeros((8, 3), dtype=torch.int8, device="cuda")
    info = torch.zeros(2, dtype=torch.int64, device="cuda")
    with pytest.raises(lib.MtpError) as e:
        lib.neighbors_build_static(pos, np.eye(3) * 200.0, 5.0, off, idx, shift, None, info)
    assert e.value.code == lib.ESIZE and "MTP_NB_STATIC_MAX_ATOMS = 32768" in str(e.value)
    with pytest.raises(lib.MtpError) as e:
        lib.neighbors_build_static(pos[:10], np.zeros((3, 3)), 5.0, off, idx, shift, None, info)
    assert e.value.code == lib.EBOX
    torch.cuda.synchronize()


def test_static_workspace_at_the_limit(lib, torch):
    """the largest system the static array takes: 32 768 atoms of the bcc lattice recipe, against the workspace path"""
    w = make_workload(1, 1)
    reps = 3                                                                     # 2 000 atoms x 16 -> cut to the limit
    pos = np.concatenate([w.pos + np.array([i, j, k]) @ w.box for i in range(reps) for j in range(reps) for k in range(reps)])
    pos = np.ascontiguousarray(pos[:lib.NB_STATIC_MAX_ATOMS])
    box = w.box * reps
    p = torch.as_tensor(pos).cuda()
    ref = lib.neighbors_build(p, box, 5.0)
    off, idx, shift, rev, info = _static(lib, torch, p, box, 5.0, ref["nnz"])
    torch.cuda.synchronize()
    n = ref["nnz"]
    assert p.shape[0] == lib.NB_STATIC_MAX_ATOMS and info.cpu().tolist() == [n, 0]
    assert torch.equal(off, ref["off"]) and torch.equal(idx, ref["idx"][:n]) and torch.equal(shift, ref["shift"][:n])
    assert torch.equal(rev, ref["rev"][:n])
