"""Plain CPU evaluation of the MTP energy / force / virial / grade.

Written from BASELINE.json north_star and SURVEY.md 8(c) steps 1-8 (PAPER.md gives no
formula; readings G1-G24 are listed in DESIGN.md).  Dense 3^nu tensors, numpy einsum,
one atom at a time, nothing blocked or fused.  `dtype` is np.float64 (the oracle) or
np.longdouble (x87 80-bit, the rounding arbiter of reading G16).

Test infrastructure only (see oracle/__init__.py); parity status: pinned by the tests
named there, "parity unpinned" against any trained-potential output.
"""
from __future__ import annotations

import dataclasses
import numpy as np

from . import basis as _basis


@dataclasses.dataclass
class Potential:
    lev_max: int
    n_mu: int
    n_beta: int
    r_min: float
    r_cut: float
    c: np.ndarray      # [S][S][n_mu][n_beta], index z_i, z_j, mu, beta   (G6)
    xi0: np.ndarray    # [S]                                            (G13, G20)
    xi: np.ndarray     # [n_basis], canonical alpha order               (G11)


# ---------------------------------------------------------------- steps 1-3: radial part
def radial_basis(r, r_min, r_cut, n_beta, dtype=np.float64):
    """Step 2: xi = (2r - R_min - R_cut)/(R_cut - R_min); T_0 = 1, T_1 = xi,
    T_{b+1} = 2 xi T_b - T_{b-1}; Q_b = T_b (R_cut - r)^2 and dQ_b/dr (step 6).
    No clamp for r < R_min (G2).  r: array [n] -> Q, dQ: [n_beta][n]."""
    r = np.asarray(r, dtype=dtype)
    r_min = dtype(r_min)
    r_cut = dtype(r_cut)
    two = dtype(2)
    x = (two * r - r_min - r_cut) / (r_cut - r_min)
    dx = two / (r_cut - r_min)
    T = [np.ones_like(r), x.copy()]
    dT = [np.zeros_like(r), np.ones_like(r)]          # d T_b / d xi
    for b in range(1, n_beta - 1):
        T.append(two * x * T[b] - T[b - 1])
        dT.append(two * T[b] + two * x * dT[b] - dT[b - 1])
    s = (r_cut - r) ** 2
    ds = -two * (r_cut - r)
    Q = np.stack([T[b] * s for b in range(n_beta)])
    dQ = np.stack([dT[b] * dx * s + T[b] * ds for b in range(n_beta)])
    return Q, dQ


def radial_functions(pot: Potential, zi: int, zj: np.ndarray, r: np.ndarray, dtype=np.float64):
    """Step 3: f_mu = sum_b c[z_i][z_j][mu][b] Q_b(r), and f'_mu.  -> [n_mu][n]."""
    Q, dQ = radial_basis(r, pot.r_min, pot.r_cut, pot.n_beta, dtype)
    cij = np.asarray(pot.c, dtype=dtype)[zi][zj]           # [n][n_mu][n_beta]
    f = np.einsum("jmb,bj->mj", cij, Q)
    df = np.einsum("jmb,bj->mj", cij, dQ)
    return f, df


# ---------------------------------------------------------------- step 4: moments
def _powers(rv: np.ndarray, nu_max: int):
    """P[nu][j] = r_j^{(x) nu} flattened to 3^nu (dense, step 4)."""
    n = rv.shape[0]
    P = [np.ones((n, 1), dtype=rv.dtype)]
    for _ in range(nu_max):
        P.append((P[-1][:, :, None] * rv[:, None, :]).reshape(n, 3 * P[-1].shape[1]))
    return P


def moments(pot: Potential, f: np.ndarray, rv: np.ndarray):
    """M_{mu,nu} = sum_j f_mu(r_j) r_j^{(x) nu}, dense arrays of shape (3,)*nu."""
    labels = _basis.moment_labels(pot.lev_max)
    nu_max = max(nu for _, nu in labels)
    P = _powers(rv, nu_max)
    M = {}
    for (mu, nu) in labels:
        M[(mu, nu)] = (f[mu] @ P[nu]).reshape((3,) * nu)
    return M, P


# ---------------------------------------------------------------- step 5: scalar basis
def _einsum_lists(key):
    """Index lists of a connected scalar: an edge of multiplicity k between u and v
    puts k fresh summation labels on both tensors (plain Einstein sum, G12)."""
    labels, ut = key
    n = len(labels)
    lists = [[] for _ in range(n)]
    nxt = 0
    p = 0
    for i in range(n):
        for j in range(i + 1, n):
            for _ in range(ut[p]):
                lists[i].append(nxt)
                lists[j].append(nxt)
                nxt += 1
            p += 1
    return lists


def scalar_value(key, M):
    labels, _ = key
    lists = _einsum_lists(key)
    args = []
    for (_, mu, nu), l in zip(labels, lists):
        args += [M[(mu, nu)], l]
    return np.einsum(*args, [])


def scalar_gradients(key, M):
    """d s / d M_v for every vertex v: the contraction with that tensor left out."""
    labels, _ = key
    lists = _einsum_lists(key)
    n = len(labels)
    out = []
    for v in range(n):
        if n == 1:
            out.append(np.ones((), dtype=M[(labels[0][1], labels[0][2])].dtype))
            continue
        args = []
        for w in range(n):
            if w != v:
                args += [M[(labels[w][1], labels[w][2])], lists[w]]
        out.append(np.einsum(*args, lists[v]))
    return out


def basis_values(pot: Potential, M):
    """B_alpha for all alpha in canonical order, plus the connected-scalar values."""
    comps = _basis.connected_scalars(pot.lev_max)
    s = {k: scalar_value(k, M) for k in comps}
    funcs = _basis.basis_functions(pot.lev_max)
    dt = next(iter(M.values())).dtype
    B = np.empty(len(funcs), dtype=dt)
    for a, func in enumerate(funcs):
        v = dt.type(1)
        for k in func:
            v = v * s[k]
        B[a] = v
    return B, s


# ---------------------------------------------------------------- steps 5-6: one atom
def atom_eval(pot: Potential, zi: int, rv: np.ndarray, zj: np.ndarray, dtype=np.float64,
              want_grad: bool = True):
    """E_i, B(n_i) and d_ij = dE_i/dr_ij for the listed neighbour vectors rv [n][3].
    Neighbours with |r| >= R_cut contribute exactly nothing (G3)."""
    rv = np.asarray(rv, dtype=dtype).reshape(-1, 3)
    zj = np.asarray(zj, dtype=np.int64).reshape(-1)
    n_all = rv.shape[0]
    r_all = np.sqrt((rv ** 2).sum(axis=1))
    keep = r_all < dtype(pot.r_cut)
    rv_k, zj_k, r = rv[keep], zj[keep], r_all[keep]
    f, df = radial_functions(pot, zi, zj_k, r, dtype)
    M, P = moments(pot, f, rv_k)
    B, s = basis_values(pot, M)
    xi = np.asarray(pot.xi, dtype=dtype)
    E_i = dtype(pot.xi0[zi]) + (xi * B).sum()
    d = np.zeros((n_all, 3), dtype=dtype)
    if not want_grad:
        return E_i, B, d
    # dE/ds_k by the product rule over the functions
    funcs = _basis.basis_functions(pot.lev_max)
    sbar = {k: dtype(0) for k in s}
    for a, func in enumerate(funcs):
        for p, k in enumerate(func):
            w = xi[a]
            for q, k2 in enumerate(func):
                if q != p:
                    w = w * s[k2]
            sbar[k] = sbar[k] + w
    # G_{mu,nu} = dE_i/dM_{mu,nu}  (dense, every slot independent)
    G = {lab: np.zeros((3,) * lab[1], dtype=dtype) for lab in M}
    for k, grads in ((k, scalar_gradients(k, M)) for k in s):
        for (_, mu, nu), g in zip(k[0], grads):
            G[(mu, nu)] = G[(mu, nu)] + sbar[k] * g
    # chain rule through step 4: dM/dr_j = f' rhat (x) r^nu + f sum_slots r^(nu-1) (x) e
    dk = np.zeros((rv_k.shape[0], 3), dtype=dtype)
    rhat = rv_k / r[:, None]
    for (mu, nu), g in G.items():
        radial_part = P[nu] @ g.reshape(-1)                      # <G, r^nu>        [n]
        dk += (df[mu] * radial_part)[:, None] * rhat
        for slot in range(nu):
            gs = np.moveaxis(g, slot, 0).reshape(3, -1)         # [3][3^(nu-1)]
            dk += f[mu][:, None] * (P[nu - 1] @ gs.T)
    d[keep] = dk
    return E_i, B, d


# ---------------------------------------------------------------- step 1 + 7: configuration
def pair_vectors(i, pos, box, off, idx, shift=None):
    """Step 1: r_ij = x_j - x_i + s.box for the CSR row of atom i.  With shift=None the
    minimum image is used (G17; legal only when every box height exceeds 2 R_cut)."""
    js = idx[off[i]:off[i + 1]]
    d = pos[js] - pos[i]
    if shift is not None:
        d = d + shift[off[i]:off[i + 1]].astype(pos.dtype) @ box
    else:
        frac = d @ np.linalg.inv(box)
        d = d - np.round(frac) @ box
    return js, d


def evaluate(pot: Potential, pos, types, box, off, idx, shift=None, dtype=np.float64,
             atoms=None, want_grad=True):
    """Steps 1-7 over a configuration.  Returns dict with E, E_i [N], F [N][3],
    W [3][3] (W_ab = -sum r_a d_b, eV), B [N][n_basis], d [nnz][3].
    `atoms`: optional subset of centre atoms (then E, F, W only hold their share)."""
    pos = np.asarray(pos, dtype=dtype)
    box = np.asarray(box, dtype=dtype)
    n = pos.shape[0]
    todo = range(n) if atoms is None else atoms
    n_basis = len(_basis.basis_functions(pot.lev_max))
    E_i = np.zeros(n, dtype=dtype)
    F = np.zeros((n, 3), dtype=dtype)
    W = np.zeros((3, 3), dtype=dtype)
    B = np.zeros((n, n_basis), dtype=dtype)
    d_all = np.zeros((idx.shape[0], 3), dtype=dtype)
    for i in todo:
        js, rv = pair_vectors(i, pos, box, off, idx, shift)
        e, b, d = atom_eval(pot, int(types[i]), rv, types[js], dtype, want_grad)
        E_i[i] = e
        B[i] = b
        d_all[off[i]:off[i + 1]] = d
        for p, j in enumerate(js):               # step 7
            F[i] += d[p]
            F[j] -= d[p]
        W -= rv.T @ d
    return dict(E=E_i.sum(), E_i=E_i, F=F, W=W, B=B, d=d_all)


def virial6(W):
    """Order xx, yy, zz, xy, xz, yz (G18)."""
    return np.array([W[0, 0], W[1, 1], W[2, 2], W[0, 1], W[0, 2], W[1, 2]])


# ---------------------------------------------------------------- step 8: grades
def grade_neighbourhood(B, Ainv):
    """gamma_i = max_k | sum_alpha B_alpha(n_i) Ainv[alpha][k] |."""
    return np.abs(np.asarray(B) @ np.asarray(Ainv, dtype=B.dtype)).max(axis=1)


def grade_configuration(B, Ainv):
    """gamma = max_k | (sum_i B(n_i)) Ainv |_k."""
    Bsum = np.asarray(B).sum(axis=0)
    return np.abs(Bsum @ np.asarray(Ainv, dtype=B.dtype)).max(), Bsum


# ---------------------------------------------------------------- own neighbour search
def brute_force_neighbours(pos, box, r_cut, rows=None):
    """The oracle's own O(27 N^2) search (north_star: 'brute-force neighbor search on
    small inputs'); returns CSR (off, idx, shift), rows ordered by (j, shift).
    `rows`: only these centre atoms (the CSR then has len(rows) rows, in that order)."""
    pos = np.asarray(pos, dtype=np.float64)
    n = pos.shape[0]
    off, idx, sh = [0], [], []
    for i in (range(n) if rows is None else rows):
        row = []
        for j in range(n):
            for sx in (-1, 0, 1):
                for sy in (-1, 0, 1):
                    for sz in (-1, 0, 1):
                        if i == j and sx == 0 and sy == 0 and sz == 0:
                            continue
                        v = pos[j] - pos[i] + sx * box[0] + sy * box[1] + sz * box[2]
                        if v @ v < r_cut * r_cut:
                            row.append((j, sx, sy, sz))
        row.sort()
        idx += [e[0] for e in row]
        sh += [e[1:] for e in row]
        off.append(len(idx))
    return (np.array(off, np.int64), np.array(idx, np.int32),
            np.array(sh, np.int8).reshape(-1, 3))
