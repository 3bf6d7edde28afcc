"""Synthetic workloads shaped like the paper's.

BASELINE.json `configs[0..4]` -> CONFIGS[0..4].  Seeds: 251000193 + config index
(SURVEY.md 8(c) G23).  Draw order is fixed: positions, species, c, xi0, xi, then
(config 5) the active-set factors.  Everything here is input preparation; the
MTP arithmetic lives in `oracle/` (CPU) and `paper_2510_00193_b200/csrc` (CUDA).
"""
from __future__ import annotations

import dataclasses
import numpy as np

BASE_SEED = 251000193

# name, lattice, cells per side, lattice constant (A), sigma (A), species fractions,
# lev_max, n_mu (number of radial functions the level uses), grade requested
CONFIGS = [
    dict(name="c1_bcc4_lev10", lattice="bcc", cells=4, a=2.87, sigma=0.05,
         fractions=(1.0,), lev_max=10, n_mu=3, grade=False),
    dict(name="c2_bcc10_lev16", lattice="bcc", cells=10, a=2.87, sigma=0.10,
         fractions=(1.0,), lev_max=16, n_mu=4, grade=False),
    dict(name="c3_bcc30_lev20", lattice="bcc", cells=30, a=2.87, sigma=0.10,
         fractions=(0.5, 0.5), lev_max=20, n_mu=5, grade=False),
    dict(name="c4_fcc64_lev16", lattice="fcc", cells=64, a=3.6, sigma=0.10,
         fractions=(0.5, 0.3, 0.2), lev_max=16, n_mu=4, grade=False),
    dict(name="c5_bcc50_lev24", lattice="bcc", cells=50, a=2.87, sigma=0.15,
         fractions=(0.5, 0.5), lev_max=24, n_mu=6, grade=True),
]
R_MIN = 2.0
R_CUT = 5.0
N_BETA = 8

_BASIS = {
    "bcc": np.array([[0.0, 0.0, 0.0], [0.5, 0.5, 0.5]]),
    "fcc": np.array([[0.0, 0.0, 0.0], [0.5, 0.5, 0.0], [0.5, 0.0, 0.5], [0.0, 0.5, 0.5]]),
    "sc": np.array([[0.0, 0.0, 0.0]]),
}


@dataclasses.dataclass
class Workload:
    name: str
    lev_max: int
    n_mu: int
    n_beta: int
    r_min: float
    r_cut: float
    n_species: int
    box: np.ndarray        # [3][3] rows = lattice vectors (orthorhombic here)
    pos: np.ndarray        # [N][3] f64, wrapped into the box
    types: np.ndarray      # [N] i32
    c: np.ndarray          # [S][S][n_mu][n_beta] f64, index z_i, z_j, mu, beta
    xi0: np.ndarray        # [S] f64
    xi: np.ndarray         # [n_basis] f64
    off: np.ndarray        # [N+1] i64 CSR offsets (full list)
    idx: np.ndarray        # [nnz] i32, ascending j inside a row
    shift: np.ndarray      # [nnz][3] i8 image shift s: r_ij = x_j - x_i + s.box
    rev: np.ndarray | None  # [nnz] i32: rev[p] = CSR position of (j,i) for p=(i,j)
    Ainv: np.ndarray | None = None  # [n_basis][n_basis] row-major [alpha][k]
    seed: int = 0

    @property
    def n_atoms(self) -> int:
        return int(self.pos.shape[0])

    @property
    def nnz(self) -> int:
        return int(self.idx.shape[0])


def _lattice_sites(lattice: str, cells: int, a: float):
    basis = _BASIS[lattice]
    nb = basis.shape[0]
    g = np.arange(cells)
    ix, iy, iz = np.meshgrid(g, g, g, indexing="ij")
    cell = np.stack([ix.ravel(), iy.ravel(), iz.ravel()], axis=1)           # [C][3]
    ideal = (cell[:, None, :] + basis[None, :, :]).reshape(-1, 3) * a       # [C*nb][3]
    return ideal, nb


def neighbor_list_stencil(lattice: str, cells: int, a: float, disp: np.ndarray, r_cut: float,
                          chunk: int = 1 << 18):
    """Exact full neighbour list of a perturbed lattice.

    Atom n sits at ideal site n plus `disp[n]`.  Any pair closer than r_cut has an
    ideal separation <= r_cut + 2*max|disp|, so scanning that lattice stencil is exact.
    Returns (off i64 [N+1], idx i32 [nnz] ascending per row, shift i8 [nnz][3]); the
    shift is relative to positions wrapped into [0, L).
    """
    basis = _BASIS[lattice]
    nb = basis.shape[0]
    n = cells ** 3 * nb
    L = cells * a
    dmax = float(np.sqrt((disp ** 2).sum(axis=1)).max()) if n else 0.0
    reach = r_cut + 2.0 * dmax + 1e-9
    if reach >= L:  # the stencil would alias an atom with its own image more than once
        raise ValueError("box too small for the stencil neighbour search")
    m = int(np.ceil(reach / a)) + 1
    rng_ = np.arange(-m, m + 1)
    sten = []  # (b_from, dx, dy, dz, b_to, ideal offset vector)
    for b0 in range(nb):
        for dx in rng_:
            for dy in rng_:
                for dz in rng_:
                    for b1 in range(nb):
                        v = (np.array([dx, dy, dz]) + basis[b1] - basis[b0]) * a
                        d = float(np.sqrt((v ** 2).sum()))
                        if 0.0 < d <= reach:
                            sten.append((b0, dx, dy, dz, b1, v))
    per_b = [[s for s in sten if s[0] == b0] for b0 in range(nb)]
    ns = max(len(p) for p in per_b)
    wrapped_shift = _wrap_shift(lattice, cells, a, disp)  # [N][3] integer image each atom was wrapped by

    counts = np.zeros(n, dtype=np.int64)
    rows_j, rows_s = [], []
    SENT = np.iinfo(np.int64).max
    for lo in range(0, n, chunk):
        hi = min(n, lo + chunk)
        ids = np.arange(lo, hi)
        b_i = ids % nb
        cidx = ids // nb
        cz = cidx % cells
        cy = (cidx // cells) % cells
        cx = cidx // (cells * cells)
        key = np.full((hi - lo, ns), SENT, dtype=np.int64)   # j * 27 + shift code, sortable by j
        for b0 in range(nb):
            sel = np.nonzero(b_i == b0)[0]
            if sel.size == 0:
                continue
            for k, (_, dx, dy, dz, b1, v) in enumerate(per_b[b0]):
                jx = cx[sel] + dx
                jy = cy[sel] + dy
                jz = cz[sel] + dz
                sx, sy, sz = jx // cells, jy // cells, jz // cells    # lattice image of the site
                j = (((jx % cells) * cells + (jy % cells)) * cells + (jz % cells)) * nb + b1
                r = v[None, :] + disp[j] - disp[ids[sel]]
                ok = (r ** 2).sum(axis=1) < r_cut * r_cut
                # image shift relative to wrapped coordinates
                s = np.stack([sx, sy, sz], axis=1) + wrapped_shift[j] - wrapped_shift[ids[sel]]
                code = (s[:, 0] + 1) * 9 + (s[:, 1] + 1) * 3 + (s[:, 2] + 1)
                if ok.any() and (np.abs(s[ok]).max() > 1):
                    raise ValueError("image shift outside [-1,1]")
                kk = np.where(ok, j.astype(np.int64) * 27 + code, SENT)
                key[sel, k] = kk
        key.sort(axis=1)
        valid = key != SENT
        counts[lo:hi] = valid.sum(axis=1)
        flat = key[valid]
        rows_j.append((flat // 27).astype(np.int32))
        code = (flat % 27).astype(np.int64)
        sh = np.stack([code // 9 - 1, (code // 3) % 3 - 1, code % 3 - 1], axis=1).astype(np.int8)
        rows_s.append(sh)
    off = np.zeros(n + 1, dtype=np.int64)
    np.cumsum(counts, out=off[1:])
    idx = np.concatenate(rows_j) if rows_j else np.zeros(0, np.int32)
    shift = np.concatenate(rows_s) if rows_s else np.zeros((0, 3), np.int8)
    return off, idx, shift


def _wrap_shift(lattice, cells, a, disp):
    """Integer image w such that wrapped = ideal + disp - w*L lies in [0, L)."""
    ideal, _ = _lattice_sites(lattice, cells, a)
    L = cells * a
    return np.floor((ideal + disp) / L).astype(np.int64)


def neighbor_list_bruteforce(pos: np.ndarray, box: np.ndarray, r_cut: float):
    """O(N^2 * 27) full list for small inputs: every image s in {-1,0,1}^3 with
    |x_j - x_i + s.box| < r_cut (i==j allowed only for s != 0)."""
    n = pos.shape[0]
    imgs = np.array([[a, b, c] for a in (-1, 0, 1) for b in (-1, 0, 1) for c in (-1, 0, 1)])
    off = [0]
    idx, shift = [], []
    for i in range(n):
        ent = []
        for s in imgs:
            d = pos - pos[i] + s @ box
            r2 = (d ** 2).sum(axis=1)
            ok = r2 < r_cut * r_cut
            if not s.any():
                ok[i] = False
            for j in np.nonzero(ok)[0]:
                ent.append((int(j), int(s[0]), int(s[1]), int(s[2])))
        ent.sort()
        for e in ent:
            idx.append(e[0])
            shift.append(e[1:])
        off.append(len(idx))
    return (np.array(off, dtype=np.int64), np.array(idx, dtype=np.int32),
            np.array(shift, dtype=np.int8).reshape(-1, 3))


def reverse_index(off: np.ndarray, idx: np.ndarray, shift: np.ndarray | None = None) -> np.ndarray:
    """rev[p] = CSR position of the pair (j,i,-s) for p = (i,j,s)."""
    n = off.shape[0] - 1
    nnz = idx.shape[0]
    i_of = np.repeat(np.arange(n, dtype=np.int64), np.diff(off))
    j_of = idx.astype(np.int64)
    if shift is None:
        code = np.zeros(nnz, dtype=np.int64)
        rcode = code
    else:
        s = shift.astype(np.int64)
        code = (s[:, 0] + 1) * 9 + (s[:, 1] + 1) * 3 + (s[:, 2] + 1)
        rcode = (1 - s[:, 0]) * 9 + (1 - s[:, 1]) * 3 + (1 - s[:, 2])
    key = (i_of * n + j_of) * 27 + code
    want = (j_of * n + i_of) * 27 + rcode
    order = np.argsort(key, kind="stable")
    pos_in_sorted = np.searchsorted(key[order], want)
    if nnz and (pos_in_sorted.max() >= nnz or not np.array_equal(key[order][pos_in_sorted], want)):
        raise ValueError("neighbour list is not symmetric")
    return order[pos_in_sorted].astype(np.int32)


def active_set_inverse(rng: np.random.Generator, n: int) -> np.ndarray:
    """BASELINE.json configs[4]: A = Q diag(d), Q from QR of a Gaussian, d ~ U[0.5,2];
    returns A^{-1} = diag(1/d) Q^T, row-major [alpha][k]."""
    g = rng.standard_normal((n, n))
    q, _ = np.linalg.qr(g)
    d = rng.uniform(0.5, 2.0, size=n)
    return np.ascontiguousarray((q.T) / d[:, None])


def make_workload(config: int | dict, n_basis: int, cells: int | None = None,
                  with_rev: bool = True, with_ainv: bool | None = None,
                  seed: int | None = None) -> Workload:
    """Build configs[config] (0-based).  `cells` overrides the lattice repeat count to
    get a scaled-down instance with the same structure (parity-test sizes).  `n_basis`
    (length of xi, size of A) comes from the caller's basis enumeration."""
    if isinstance(config, dict):
        cfg, ci = dict(config), int(config.get("index", 0))
    else:
        cfg, ci = dict(CONFIGS[config]), int(config)
    if cells is not None:
        cfg["cells"] = cells
    seed = BASE_SEED + ci if seed is None else seed
    rng = np.random.default_rng(seed)
    ideal, nb = _lattice_sites(cfg["lattice"], cfg["cells"], cfg["a"])
    n = ideal.shape[0]
    L = cfg["cells"] * cfg["a"]
    disp = rng.normal(0.0, cfg["sigma"], size=(n, 3))
    pos = ideal + disp
    pos -= np.floor(pos / L) * L
    fr = np.asarray(cfg["fractions"], dtype=np.float64)
    S = fr.shape[0]
    types = rng.choice(S, size=n, p=fr / fr.sum()).astype(np.int32) if S > 1 else np.zeros(n, np.int32)
    n_mu = cfg["n_mu"]
    c = rng.uniform(-0.1, 0.1, size=(S, S, n_mu, N_BETA))
    xi0 = rng.uniform(-0.1, 0.1, size=S)
    xi = rng.uniform(-0.1, 0.1, size=n_basis)
    off, idx, shift = neighbor_list_stencil(cfg["lattice"], cfg["cells"], cfg["a"], disp, R_CUT)
    rev = reverse_index(off, idx, shift) if with_rev else None
    want_a = cfg["grade"] if with_ainv is None else with_ainv
    Ainv = active_set_inverse(rng, n_basis) if want_a else None
    return Workload(name=cfg["name"], lev_max=cfg["lev_max"], n_mu=n_mu, n_beta=N_BETA,
                    r_min=R_MIN, r_cut=R_CUT, n_species=S, box=np.eye(3) * L, pos=pos,
                    types=types, c=c, xi0=xi0, xi=xi, off=off, idx=idx, shift=shift, rev=rev,
                    Ainv=Ainv, seed=seed)


def random_cluster(seed: int, n_atoms: int, box_len: float, n_species: int = 1,
                   r_min_sep: float = 1.6):
    """Non-lattice test input: random positions in a cubic periodic box with a minimum
    separation (rejection sampling); used by oracle pins and edge-case parity tests."""
    rng = np.random.default_rng(seed)
    pts = []
    box = np.eye(3) * box_len
    tries = 0
    while len(pts) < n_atoms and tries < 100000:
        tries += 1
        p = rng.uniform(0, box_len, size=3)
        ok = True
        for q in pts:
            d = p - q
            d -= np.round(d / box_len) * box_len
            if (d ** 2).sum() < r_min_sep ** 2:
                ok = False
                break
        if ok:
            pts.append(p)
    pos = np.array(pts).reshape(-1, 3)
    types = rng.integers(0, n_species, size=pos.shape[0]).astype(np.int32)
    return pos, types, box
