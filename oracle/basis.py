"""Oracle-side enumeration of the MTP scalar basis from the level rule.

Follows BASELINE.json north_star ("B_alpha as a contraction ... over products of M
with level lev(M_{mu,nu}) = 2+4mu+nu summed <= lev_max") with the readings G8, G9,
G11 of SURVEY.md 8(c) (restated in DESIGN.md):

* a *connected scalar* is either one vertex M_{mu,0}, or a connected loop-free
  multigraph whose vertex v carries a label (mu_v, nu_v), nu_v >= 1, and has degree
  nu_v (an edge of multiplicity k contracts k index pairs);
* a *basis function* is a multiset of connected scalars (their product) whose levels
  sum to <= lev_max;
* canonical key of a connected scalar: (labels, adjacency) with labels the tuple of
  (lev, mu, nu) sorted ascending and adjacency the lexicographically smallest
  upper-triangular tuple (k01, k02, ..., k12, ...) over vertex orders that keep the
  label tuple sorted;
* canonical key of a function: the ascending tuple of its component keys; functions
  are ordered by (total level, number of components, key).

Test infrastructure only (see oracle/__init__.py).
"""
from __future__ import annotations

import itertools
from functools import lru_cache


def lev_of(mu: int, nu: int) -> int:
    return 2 + 4 * mu + nu


def moment_labels(lev_max: int):
    """(mu, nu) of every moment tensor that can occur in a scalar of level <= lev_max
    (SURVEY.md 8(c) step 4 / G8): nu = 0 needs lev <= lev_max; nu >= 1 needs a partner
    carrying at least nu indices, cheapest partner M_{0,nu}: 2*lev... = 4+4mu+2nu."""
    out = []
    mu = 0
    while lev_of(mu, 0) <= lev_max:
        nu = 0
        while True:
            ok = lev_of(mu, 0) <= lev_max if nu == 0 else (4 * mu + 2 * nu <= lev_max - 4)
            if not ok:
                break
            out.append((mu, nu))
            nu += 1
        mu += 1
    return out


def _adjacencies(nus):
    """All symmetric zero-diagonal non-negative integer matrices with row sums nus,
    as upper-triangular tuples in row-major order."""
    n = len(nus)
    pairs = [(i, j) for i in range(n) for j in range(i + 1, n)]
    res = []

    def rec(p, rem, cur):
        if p == len(pairs):
            if all(r == 0 for r in rem):
                res.append(tuple(cur))
            return
        i, j = pairs[p]
        # last pair of row i must use up the remainder of row i
        last_of_row_i = (j == n - 1)
        hi = min(rem[i], rem[j])
        lo = rem[i] if last_of_row_i else 0
        if lo > hi:
            return
        for k in range(lo, hi + 1):
            rem[i] -= k
            rem[j] -= k
            cur.append(k)
            rec(p + 1, rem, cur)
            cur.pop()
            rem[i] += k
            rem[j] += k

    rec(0, list(nus), [])
    return res


def _matrix(n, ut):
    a = [[0] * n for _ in range(n)]
    p = 0
    for i in range(n):
        for j in range(i + 1, n):
            a[i][j] = a[j][i] = ut[p]
            p += 1
    return a


def _connected(n, a):
    seen = {0}
    stack = [0]
    while stack:
        u = stack.pop()
        for v in range(n):
            if a[u][v] and v not in seen:
                seen.add(v)
                stack.append(v)
    return len(seen) == n


def _canonical_adjacency(labels, a):
    """Smallest upper-triangular tuple over permutations that only exchange vertices
    with identical labels (labels is already sorted)."""
    n = len(labels)
    groups = []
    i = 0
    while i < n:
        j = i
        while j < n and labels[j] == labels[i]:
            j += 1
        groups.append(list(range(i, j)))
        i = j
    best = None
    for perm_parts in itertools.product(*[itertools.permutations(g) for g in groups]):
        perm = [v for part in perm_parts for v in part]
        ut = tuple(a[perm[i]][perm[j]] for i in range(n) for j in range(i + 1, n))
        if best is None or ut < best:
            best = ut
    return best


@lru_cache(maxsize=None)
def connected_scalars(lev_max: int):
    """Sorted list of canonical keys of all connected scalars with level <= lev_max.
    key = (labels, adjacency); labels = ((lev, mu, nu), ...)."""
    keys = set()
    mu = 0
    while lev_of(mu, 0) <= lev_max:
        keys.add((((lev_of(mu, 0), mu, 0),), ()))
        mu += 1
    types = []  # vertex types with nu >= 1, sorted by (lev, mu, nu)
    for mu in range(0, lev_max):
        for nu in range(1, lev_max):
            if lev_of(mu, nu) <= lev_max:
                types.append((lev_of(mu, nu), mu, nu))
    types.sort()

    def rec(start, chosen, total):
        n = len(chosen)
        if n >= 2:
            nus = [t[2] for t in chosen]
            s = sum(nus)
            if s % 2 == 0 and 2 * max(nus) <= s and s >= 2 * (n - 1):
                labels = tuple(chosen)
                for ut in _adjacencies(nus):
                    a = _matrix(n, ut)
                    if _connected(n, a):
                        keys.add((labels, _canonical_adjacency(labels, a)))
        for t in range(start, len(types)):
            if total + types[t][0] <= lev_max:
                chosen.append(types[t])
                rec(t, chosen, total + types[t][0])
                chosen.pop()

    rec(0, [], 0)
    return sorted(keys)


def component_level(key) -> int:
    return sum(l[0] for l in key[0])


@lru_cache(maxsize=None)
def basis_functions(lev_max: int):
    """Canonical ordered list of basis functions; each is a tuple of component keys."""
    comps = connected_scalars(lev_max)
    levs = [component_level(k) for k in comps]
    out = []

    def rec(start, chosen, total):
        if chosen:
            out.append((total, len(chosen), tuple(chosen)))
        for t in range(start, len(comps)):
            if total + levs[t] <= lev_max:
                chosen.append(comps[t])
                rec(t, chosen, total + levs[t])
                chosen.pop()

    rec(0, [], 0)
    out.sort()
    return [f[2] for f in out]


def describe(func) -> list:
    """Flat integer description of a function, the form in which the CUDA library's
    enumerator exports its list (include/mtp_b200.h `basis_desc`): n_components, then
    per component n_vertices, (mu, nu) per vertex, upper-triangular adjacency."""
    d = [len(func)]
    for labels, ut in func:
        d.append(len(labels))
        for (_, mu, nu) in labels:
            d += [mu, nu]
        d += list(ut)
    return d
