"""Shared helpers for the parity tests: build the oracle potential and the CUDA potential
from the same seeded workload (workloads/ holds no method arithmetic)."""
import numpy as np

from oracle import basis as obasis
from oracle import mtp as omtp


def n_basis_of(lev):
    return len(obasis.basis_functions(lev))


def oracle_pot(w):
    return omtp.Potential(w.lev_max, w.n_mu, w.n_beta, w.r_min, w.r_cut, w.c, w.xi0, w.xi)


def gpu_pot(lib, w, table=None):
    table = lib.Table(w.lev_max) if table is None else table
    return lib.Potential(table, w.n_species, w.n_beta, w.r_min, w.r_cut, w.c, w.xi0, w.xi)


def to_dev(w, torch, with_shift=True):
    dev = torch.device("cuda:0")
    t = lambda a, dt: torch.as_tensor(np.ascontiguousarray(a), dtype=dt).to(dev)
    return dict(pos=t(w.pos, torch.float64), types=t(w.types, torch.int32), off=t(w.off, torch.int64),
                idx=t(w.idx, torch.int32), shift=t(w.shift, torch.int8) if with_shift else None,
                rev=t(w.rev, torch.int32) if w.rev is not None else None)


def scales(pot, out, off, idx):
    """G16 scales: s_E,i = max(1, sum_a |xi_a B_a|), s_F,k = max(1, sum_j |d_kj| + |d_jk|)."""
    sE = np.maximum(1.0, np.abs(out["B"] * pot.xi[None, :]).sum(axis=1))
    n = out["F"].shape[0]
    sF = np.zeros(n)
    dn = np.abs(out["d"]).sum(axis=1)
    i_of = np.repeat(np.arange(n), np.diff(off))
    np.add.at(sF, i_of, dn)
    np.add.at(sF, idx, dn)
    return sE, np.maximum(1.0, sF)
