"""Thin ctypes binding of include/mtp_b200.h -- argument marshalling only.

Every numeric step runs in libmtp_b200.so's CUDA kernels; PyTorch is used for device
memory and streams.  There is no CPU fallback: if the shared library is missing (and
cannot be built) importing this module raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmtp_b200.so")

OK, EINVAL, ESIZE, EBOX, ECUDA, EUNSUP, ENOMEM = 0, -1, -2, -3, -4, -5, -6
OPT_CHUNK_ATOMS, OPT_FORCE_MODE, OPT_VARIANT, OPT_PROFILE, OPT_TREE_CODEGEN, OPT_CHUNK_PAIRS, OPT_SKIN_LIST = 1, 2, 3, 4, 5, 6, 7
INFO_TREE_KERNELS, INFO_TREE_PROGRAMS, INFO_INPUT_ERRORS, INFO_SCRATCH_OVERFLOW = 100, 101, 102, 103
FORCE_GATHER, FORCE_ATOMIC, FORCE_AUTO = 0, 1, 2
VARIANT_AUTO, VARIANT_THREAD, VARIANT_BLOCK = 0, 1, 2

_I32P = C.POINTER(C.c_int32)


class MtpParams(C.Structure):
    _fields_ = [
        ("n_species", C.c_int32), ("n_radial_basis", C.c_int32), ("n_radial_funcs", C.c_int32),
        ("r_min", C.c_double), ("r_cut", C.c_double), ("lev_max", C.c_int32),
        ("n_basic", C.c_int32), ("basic", _I32P), ("n_nodes", C.c_int32), ("n_prod", C.c_int32),
        ("prod", _I32P), ("n_basis", C.c_int32), ("basis_node", _I32P),
        ("c", C.POINTER(C.c_double)), ("xi0", C.POINTER(C.c_double)), ("xi", C.POINTER(C.c_double)),
        ("n_desc", C.c_int32), ("basis_desc", _I32P), ("basis_desc_off", _I32P),
    ]


class AlPolicy(C.Structure):
    """mtp_al_policy of include/mtp_b200.h"""
    _fields_ = [("grade_every", C.c_int32), ("mode", C.c_int32), ("select_threshold", C.c_double),
                ("break_threshold", C.c_double), ("max_selected", C.c_int32)]


EXPORTS = ["mtp_enumerate", "mtp_table_free", "mtp_create", "mtp_destroy", "mtp_last_error",
           "mtp_set_option", "mtp_get_option", "mtp_workspace_bytes", "mtp_compute", "mtp_grade",
           "mtp_compute_host", "mtp_debug_moments", "mtp_launch_count", "mtp_peak_dfma",
           "mtp_cost_model", "mtp_profile_read", "mtp_table_plan", "mtp_k2_program",
           "mtp_neighbors_workspace_bytes", "mtp_neighbors_build", "mtp_neighbors_build_static",
           "mtp_md_al_workspace_bytes", "mtp_md_run_al", "mtp_graph_capture", "mtp_graph_launch", "mtp_graph_destroy", "mtp_rows_workspace_bytes", "mtp_compute_rows", "mtp_grade_rows", "mtp_grade_cfg_from_sum", "mtp_md_workspace_bytes", "mtp_md_run",
           "mtp_compute_host_pos"]


def _build():
    import importlib.util
    spec = importlib.util.spec_from_file_location("_mtp_b200_build", os.path.join(_HERE, "build.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    mod.build()


def _load():
    if not os.path.exists(LIB_PATH):
        _build()
    lib = C.CDLL(LIB_PATH)
    if not all(hasattr(lib, name) for name in EXPORTS):      # stale build: rebuild once, then insist
        _build()
        lib = C.CDLL(LIB_PATH)
        if not all(hasattr(lib, name) for name in EXPORTS):
            raise ImportError("%s is stale (missing exports): run `python paper_2510_00193_b200/build.py`" % LIB_PATH)
    vp, i64, dbl = C.c_void_p, C.c_int64, C.c_double
    lib.mtp_enumerate.argtypes = [C.c_int32, C.POINTER(MtpParams)]
    lib.mtp_table_free.argtypes = [C.POINTER(MtpParams)]
    lib.mtp_table_free.restype = None
    lib.mtp_create.argtypes = [C.POINTER(vp), C.POINTER(MtpParams)]
    lib.mtp_destroy.argtypes = [vp]
    lib.mtp_destroy.restype = None
    lib.mtp_last_error.argtypes = [vp]
    lib.mtp_last_error.restype = C.c_char_p
    lib.mtp_set_option.argtypes = [vp, C.c_int, i64]
    lib.mtp_get_option.argtypes = [vp, C.c_int, C.POINTER(i64)]
    lib.mtp_workspace_bytes.argtypes = [vp, i64, i64, C.c_int, C.POINTER(C.c_size_t)]
    lib.mtp_compute.argtypes = [vp, i64, vp, vp, C.POINTER(dbl), vp, vp, vp, vp, i64, vp, vp, vp, vp, vp,
                                C.c_size_t, vp]
    lib.mtp_grade.argtypes = [vp, i64, vp, vp, C.POINTER(dbl), vp, vp, vp, i64, vp, C.c_int, vp, vp, vp, vp,
                              vp, C.c_size_t, vp]
    lib.mtp_compute_host.argtypes = [vp, i64, vp, vp, C.POINTER(dbl), vp, vp, vp, vp, i64, vp, vp, vp, vp]
    lib.mtp_debug_moments.argtypes = [vp, i64, vp, vp, C.POINTER(dbl), vp, vp, vp, vp, vp, vp, vp, C.c_size_t, vp]
    lib.mtp_launch_count.restype = i64
    lib.mtp_peak_dfma.argtypes = [i64, vp, C.POINTER(dbl), vp]
    lib.mtp_cost_model.argtypes = [vp, C.POINTER(dbl), C.POINTER(dbl), C.POINTER(dbl)]
    lib.mtp_profile_read.argtypes = [vp, C.POINTER(dbl), C.POINTER(i64)]
    lib.mtp_table_plan.argtypes = [C.POINTER(MtpParams), C.POINTER(i64)]
    lib.mtp_neighbors_workspace_bytes.argtypes = [i64, C.POINTER(C.c_size_t)]
    lib.mtp_neighbors_build.argtypes = [i64, vp, C.POINTER(dbl), dbl, i64, vp, vp, vp, vp, vp, vp, C.c_size_t, vp]
    lib.mtp_graph_capture.argtypes = [vp, i64, vp, vp, C.POINTER(dbl), vp, vp, vp, vp, i64, vp, vp, vp, vp, vp, C.c_size_t, C.POINTER(vp)]
    lib.mtp_graph_launch.argtypes = [vp, vp]
    lib.mtp_graph_destroy.argtypes = [vp]
    lib.mtp_md_al_workspace_bytes.argtypes = [vp, i64, i64, C.POINTER(C.c_size_t)]
    lib.mtp_md_run_al.argtypes = [vp, i64, vp, vp, vp, C.POINTER(dbl), C.POINTER(dbl), dbl, i64, C.c_int32, dbl, i64, vp,
                                  C.POINTER(AlPolicy), vp, vp, vp, vp, vp, vp, vp, C.POINTER(i64), C.POINTER(dbl), C.POINTER(i64),
                                  C.POINTER(dbl), vp, C.c_size_t, vp]
    lib.mtp_rows_workspace_bytes.argtypes = [vp, i64, i64, i64, C.c_int, C.POINTER(C.c_size_t)]
    lib.mtp_compute_rows.argtypes = [vp, i64, vp, vp, C.POINTER(dbl), i64, i64, vp, vp, vp, i64, vp, vp, vp, vp, vp, C.c_size_t, vp]
    lib.mtp_grade_rows.argtypes = [vp, i64, vp, vp, C.POINTER(dbl), i64, i64, vp, vp, vp, i64, vp, vp, vp, vp, C.c_size_t, vp]
    lib.mtp_grade_cfg_from_sum.argtypes = [vp, vp, vp, vp, vp]
    lib.mtp_neighbors_build_static.argtypes = [i64, vp, C.POINTER(dbl), dbl, i64, vp, vp, vp, vp, vp, vp]
    lib.mtp_md_workspace_bytes.argtypes = [vp, i64, i64, C.POINTER(C.c_size_t)]
    lib.mtp_md_run.argtypes = [vp, i64, vp, vp, vp, C.POINTER(dbl), C.POINTER(dbl), dbl, i64, C.c_int32, dbl, i64,
                               vp, vp, vp, vp, vp, vp, C.c_size_t, vp]
    lib.mtp_compute_host_pos.argtypes = [vp, i64, vp, vp, C.POINTER(dbl), vp, vp, vp, vp, C.POINTER(i64)]
    lib.mtp_k2_program.argtypes = [C.POINTER(MtpParams), C.c_int, vp, i64, vp, i64, C.POINTER(i64)]
    return lib


_lib = _load()


class MtpError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("mtp_b200 error %d: %s" % (code, msg))
        self.code = code


class Table:
    """Contraction table emitted by mtp_enumerate (numpy copies of the C arrays)."""

    def __init__(self, lev_max: int):
        p = MtpParams()
        rc = _lib.mtp_enumerate(int(lev_max), C.byref(p))
        if rc != OK:
            raise MtpError(rc, "mtp_enumerate(%d)" % lev_max)
        try:
            self.lev_max = int(p.lev_max)
            self.n_mu = int(p.n_radial_funcs)
            self.n_basic, self.n_nodes, self.n_prod, self.n_basis = p.n_basic, p.n_nodes, p.n_prod, p.n_basis
            self.basic = np.ctypeslib.as_array(p.basic, (p.n_basic, 4)).copy()
            self.prod = (np.ctypeslib.as_array(p.prod, (p.n_prod, 4)).copy() if p.n_prod
                         else np.zeros((0, 4), np.int32))
            self.basis_node = np.ctypeslib.as_array(p.basis_node, (p.n_basis,)).copy()
            self.basis_desc = np.ctypeslib.as_array(p.basis_desc, (p.n_desc,)).copy()
            self.basis_desc_off = np.ctypeslib.as_array(p.basis_desc_off, (p.n_basis + 1,)).copy()
        finally:
            _lib.mtp_table_free(C.byref(p))

    def plan(self):
        """mtp_table_plan: how mtp_create will evaluate this table (host-only diagnostic)."""
        basic = np.ascontiguousarray(self.basic, dtype=np.int32)
        prod = np.ascontiguousarray(self.prod, dtype=np.int32)
        bn = np.ascontiguousarray(self.basis_node, dtype=np.int32)
        p = MtpParams()
        p.n_basic, p.basic, p.n_nodes = basic.shape[0], basic.ctypes.data_as(_I32P), int(self.n_nodes)
        p.n_prod, p.prod = prod.shape[0], prod.ctypes.data_as(_I32P)
        p.n_basis, p.basis_node = bn.shape[0], bn.ctypes.data_as(_I32P)
        out = (C.c_int64 * 8)()
        rc = _lib.mtp_table_plan(C.byref(p), out)
        if rc != OK:
            raise MtpError(rc, "mtp_table_plan")
        keys = ["partitioned", "threads_per_sm", "cut_rows", "groups", "top_ops", "group_ops", "ops_below_cut", "specialised"]
        return dict(zip(keys, [int(x) for x in out]))

    def k2_program(self, xi, kind=0):
        """mtp_k2_program: the register program of the whole table as data (host-only), for emulation in the tests.
        Returns dict(prog[n][7] int32, consts[m] f64, n_regs, n_slots)."""
        basic = np.ascontiguousarray(self.basic, dtype=np.int32)
        prod = np.ascontiguousarray(self.prod, dtype=np.int32)
        bn = np.ascontiguousarray(self.basis_node, dtype=np.int32)
        xi = np.ascontiguousarray(xi, dtype=np.float64)
        p = MtpParams()
        p.n_basic, p.basic, p.n_nodes = basic.shape[0], basic.ctypes.data_as(_I32P), int(self.n_nodes)
        p.n_prod, p.prod = prod.shape[0], prod.ctypes.data_as(_I32P)
        p.n_basis, p.basis_node = bn.shape[0], bn.ctypes.data_as(_I32P)
        p.xi = xi.ctypes.data_as(C.POINTER(C.c_double))
        info = (C.c_int64 * 4)()
        rc = _lib.mtp_k2_program(C.byref(p), int(kind), None, 0, None, 0, info)
        if rc != OK:
            raise MtpError(rc, "mtp_k2_program")
        prog = np.zeros((int(info[0]), 7), np.int32)
        consts = np.zeros(max(int(info[1]), 1), np.float64)
        rc = _lib.mtp_k2_program(C.byref(p), int(kind), C.c_void_p(prog.ctypes.data), prog.shape[0],
                                 C.c_void_p(consts.ctypes.data), consts.shape[0], info)
        if rc != OK:
            raise MtpError(rc, "mtp_k2_program")
        return dict(prog=prog, consts=consts[:int(info[1])], n_regs=int(info[2]), n_slots=int(info[3]))

    def describe(self, alpha: int):
        return list(self.basis_desc[self.basis_desc_off[alpha]:self.basis_desc_off[alpha + 1]])


def _ptr(t):
    return C.c_void_p(0 if t is None else t.data_ptr())


def _np_ptr(a):
    return C.c_void_p(0 if a is None else a.ctypes.data)


class Potential:
    """mtp_create / mtp_compute / mtp_grade behind torch device tensors."""

    def __init__(self, table: Table, n_species, n_beta, r_min, r_cut, c, xi0, xi,
                 basic=None, prod=None, basis_node=None, n_nodes=None):
        self.table = table
        basic = np.ascontiguousarray(table.basic if basic is None else basic, dtype=np.int32)
        prod = np.ascontiguousarray(table.prod if prod is None else prod, dtype=np.int32)
        basis_node = np.ascontiguousarray(table.basis_node if basis_node is None else basis_node, dtype=np.int32)
        c = np.ascontiguousarray(c, dtype=np.float64)
        xi0 = np.ascontiguousarray(xi0, dtype=np.float64)
        xi = np.ascontiguousarray(xi, dtype=np.float64)
        n_mu = c.shape[2]
        assert c.shape == (n_species, n_species, n_mu, n_beta)
        p = MtpParams()
        p.n_species, p.n_radial_basis, p.n_radial_funcs = int(n_species), int(n_beta), int(n_mu)
        p.r_min, p.r_cut, p.lev_max = float(r_min), float(r_cut), int(table.lev_max)
        p.n_basic, p.basic = basic.shape[0], basic.ctypes.data_as(_I32P)
        p.n_nodes = int(table.n_nodes if n_nodes is None else n_nodes)
        p.n_prod, p.prod = prod.shape[0], prod.ctypes.data_as(_I32P)
        p.n_basis, p.basis_node = basis_node.shape[0], basis_node.ctypes.data_as(_I32P)
        p.c = c.ctypes.data_as(C.POINTER(C.c_double))
        p.xi0 = xi0.ctypes.data_as(C.POINTER(C.c_double))
        p.xi = xi.ctypes.data_as(C.POINTER(C.c_double))
        p.n_desc, p.basis_desc, p.basis_desc_off = 0, None, None
        h = C.c_void_p()
        rc = _lib.mtp_create(C.byref(h), C.byref(p))
        if rc != OK:
            raise MtpError(rc, _lib.mtp_last_error(None).decode())
        self._h = h
        self.n_basis = int(p.n_basis)
        self.n_basic = int(p.n_basic)
        self._ws = None

    def close(self):
        if getattr(self, "_h", None):
            _lib.mtp_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc):
        if rc != OK:
            raise MtpError(rc, _lib.mtp_last_error(self._h).decode())

    def set_option(self, key, value):
        self._check(_lib.mtp_set_option(self._h, int(key), int(value)))

    def get_option(self, key):
        v = C.c_int64()
        self._check(_lib.mtp_get_option(self._h, int(key), C.byref(v)))
        return int(v.value)

    def workspace_bytes(self, n_atoms, nnz, want_grade=False):
        out = C.c_size_t()
        self._check(_lib.mtp_workspace_bytes(self._h, int(n_atoms), int(nnz), int(bool(want_grade)), C.byref(out)))
        return int(out.value)

    def cost_model(self):
        """mtp_cost_model: algorithmic flops per pair (K1, K3) and per atom (K2, K5)."""
        a, b, c = (C.c_double * 2)(), C.c_double(), C.c_double()
        self._check(_lib.mtp_cost_model(self._h, a, C.byref(b), C.byref(c)))
        return dict(flop_per_pair_k1=a[0], flop_per_pair_k3=a[1], flop_per_atom_tree=b.value, flop_per_atom_grade=c.value)

    def last_error(self):
        return _lib.mtp_last_error(self._h).decode()

    def profile_read(self):
        """dict class -> (ms, launches) since the last read (needs OPT_PROFILE = 1)."""
        ms = (C.c_double * 5)()
        n = (C.c_int64 * 5)()
        self._check(_lib.mtp_profile_read(self._h, ms, n))
        names = ["moments", "tree", "pairgrad", "gather", "grade"]
        return {k: (ms[i], int(n[i])) for i, k in enumerate(names)}

    def _workspace(self, nbytes, device):
        import torch
        if self._ws is None or self._ws.numel() < nbytes or self._ws.device != device:
            self._ws = torch.empty(int(nbytes), dtype=torch.uint8, device=device)
        return self._ws

    @staticmethod
    def _stream(stream):
        import torch
        s = torch.cuda.current_stream() if stream is None else stream
        return C.c_void_p(s.cuda_stream)

    def compute(self, pos, types, box, off, idx, shift=None, rev=None, want_ei=True, out=None, stream=None):
        """mtp_compute on torch CUDA tensors.  Returns dict(E[1], Ei[N], F[N,3], virial[6])."""
        import torch
        n, nnz, dev = int(pos.shape[0]), int(idx.shape[0]), pos.device
        assert pos.dtype == torch.float64 and types.dtype == torch.int32 and off.dtype == torch.int64
        assert idx.dtype == torch.int32 and pos.is_contiguous()
        if out is None:
            out = dict(E=torch.empty(1, dtype=torch.float64, device=dev),
                       Ei=torch.empty(n, dtype=torch.float64, device=dev) if want_ei else None,
                       F=torch.empty((n, 3), dtype=torch.float64, device=dev),
                       virial=torch.empty(6, dtype=torch.float64, device=dev))
        ws = self._workspace(self.workspace_bytes(n, nnz), dev)
        boxh = (C.c_double * 9)(*[float(x) for x in np.asarray(box, dtype=np.float64).reshape(9)])
        self._check(_lib.mtp_compute(self._h, n, _ptr(pos), _ptr(types), boxh, _ptr(off), _ptr(idx), _ptr(shift),
                                     _ptr(rev), nnz, _ptr(out["E"]), _ptr(out.get("Ei")), _ptr(out["F"]),
                                     _ptr(out["virial"]), _ptr(ws), ws.numel(), self._stream(stream)))
        return out

    def graph(self, pos, types, box, off, idx, shift=None, rev=None):
        """mtp_graph_capture of one compute call on these tensors.  Returns (ComputeGraph, out dict); graph.launch()
        re-evaluates from whatever the tensors hold.  The graph keeps its own workspace and references to the tensors."""
        import torch
        n, nnz, dev = int(pos.shape[0]), int(idx.shape[0]), pos.device
        out = dict(E=torch.empty(1, dtype=torch.float64, device=dev), Ei=torch.empty(n, dtype=torch.float64, device=dev),
                   F=torch.empty((n, 3), dtype=torch.float64, device=dev), virial=torch.empty(6, dtype=torch.float64, device=dev))
        ws = torch.empty(self.workspace_bytes(n, nnz), dtype=torch.uint8, device=dev)
        boxh = (C.c_double * 9)(*[float(x) for x in np.asarray(box, dtype=np.float64).reshape(9)])
        g = C.c_void_p()
        self._check(_lib.mtp_graph_capture(self._h, n, _ptr(pos), _ptr(types), boxh, _ptr(off), _ptr(idx), _ptr(shift), _ptr(rev),
                                           nnz, _ptr(out["E"]), _ptr(out["Ei"]), _ptr(out["F"]), _ptr(out["virial"]), _ptr(ws),
                                           ws.numel(), C.byref(g)))
        return ComputeGraph(self, g, (pos, types, off, idx, shift, rev, ws, out)), out

    def grade(self, pos, types, box, off, idx, Ainv, shift=None, mode=2, want_B=False, stream=None):
        import torch
        n, nnz, dev = int(pos.shape[0]), int(idx.shape[0]), pos.device
        out = dict(gamma_atom=torch.empty(n, dtype=torch.float64, device=dev) if mode != 1 else None,
                   gamma_cfg=torch.empty(1, dtype=torch.float64, device=dev) if mode != 0 else None,
                   Bsum=torch.empty(self.n_basis, dtype=torch.float64, device=dev),
                   B=torch.empty((n, self.n_basis), dtype=torch.float64, device=dev) if want_B else None)
        ws = self._workspace(self.workspace_bytes(n, nnz, True), dev)
        boxh = (C.c_double * 9)(*[float(x) for x in np.asarray(box, dtype=np.float64).reshape(9)])
        self._check(_lib.mtp_grade(self._h, n, _ptr(pos), _ptr(types), boxh, _ptr(off), _ptr(idx), _ptr(shift), nnz,
                                   _ptr(Ainv), int(mode), _ptr(out["gamma_atom"]), _ptr(out["gamma_cfg"]),
                                   _ptr(out["Bsum"]), _ptr(out["B"]), _ptr(ws), ws.numel(), self._stream(stream)))
        return out

    def compute_rows(self, pos, types, box, row_lo, row_hi, off, idx, shift=None, out=None, stream=None):
        """mtp_compute_rows: the rows [row_lo, row_hi) of the system (off = the window's own CSR, idx global).
        Returns dict(E[1], Ei[N], F[N,3], virial[6]) -- PARTIAL sums, to be added over the ranks."""
        import torch
        n, nnz, dev = int(pos.shape[0]), int(idx.shape[0]), pos.device
        if out is None:
            out = dict(E=torch.empty(1, dtype=torch.float64, device=dev), Ei=torch.zeros(n, dtype=torch.float64, device=dev),
                       F=torch.empty((n, 3), dtype=torch.float64, device=dev), virial=torch.empty(6, dtype=torch.float64, device=dev))
        wsb = C.c_size_t()
        self._check(_lib.mtp_rows_workspace_bytes(self._h, n, int(row_hi - row_lo), nnz, 0, C.byref(wsb)))
        ws = self._workspace(int(wsb.value), dev)
        boxh = (C.c_double * 9)(*[float(x) for x in np.asarray(box, dtype=np.float64).reshape(9)])
        self._check(_lib.mtp_compute_rows(self._h, n, _ptr(pos), _ptr(types), boxh, int(row_lo), int(row_hi), _ptr(off), _ptr(idx),
                                          _ptr(shift), nnz, _ptr(out["E"]), _ptr(out.get("Ei")), _ptr(out["F"]), _ptr(out["virial"]),
                                          _ptr(ws), ws.numel(), self._stream(stream)))
        return out

    def grade_rows(self, pos, types, box, row_lo, row_hi, off, idx, Ainv, shift=None, stream=None):
        """mtp_grade_rows: dict(gamma_atom[N] (window entries written), Bsum[n_basis] = the window's sum of B)."""
        import torch
        n, nnz, dev = int(pos.shape[0]), int(idx.shape[0]), pos.device
        out = dict(gamma_atom=torch.zeros(n, dtype=torch.float64, device=dev), Bsum=torch.empty(self.n_basis, dtype=torch.float64, device=dev))
        wsb = C.c_size_t()
        self._check(_lib.mtp_rows_workspace_bytes(self._h, n, int(row_hi - row_lo), nnz, 1, C.byref(wsb)))
        ws = self._workspace(int(wsb.value), dev)
        boxh = (C.c_double * 9)(*[float(x) for x in np.asarray(box, dtype=np.float64).reshape(9)])
        self._check(_lib.mtp_grade_rows(self._h, n, _ptr(pos), _ptr(types), boxh, int(row_lo), int(row_hi), _ptr(off), _ptr(idx),
                                        _ptr(shift), nnz, _ptr(Ainv), _ptr(out["gamma_atom"]), _ptr(out["Bsum"]), _ptr(ws), ws.numel(),
                                        self._stream(stream)))
        return out

    def grade_cfg_from_sum(self, Bsum, Ainv, stream=None):
        import torch
        g = torch.empty(1, dtype=torch.float64, device=Bsum.device)
        self._check(_lib.mtp_grade_cfg_from_sum(self._h, _ptr(Bsum), _ptr(Ainv), _ptr(g), self._stream(stream)))
        return g

    def debug_moments(self, pos, types, box, off, idx, shift=None, stream=None):
        """M, G as [n_basic][N] and B [N][n_basis] from one K1+K2 pass."""
        import torch
        n, dev = int(pos.shape[0]), pos.device
        M = torch.empty((self.n_basic, n), dtype=torch.float64, device=dev)
        G = torch.empty((self.n_basic, n), dtype=torch.float64, device=dev)
        B = torch.empty((n, self.n_basis), dtype=torch.float64, device=dev)
        saved = self.get_option(OPT_CHUNK_ATOMS)
        self.set_option(OPT_CHUNK_ATOMS, max(n, 1))
        ws = self._workspace(self.workspace_bytes(n, 0, True), dev)
        self.set_option(OPT_CHUNK_ATOMS, saved)
        boxh = (C.c_double * 9)(*[float(x) for x in np.asarray(box, dtype=np.float64).reshape(9)])
        self._check(_lib.mtp_debug_moments(self._h, n, _ptr(pos), _ptr(types), boxh, _ptr(off), _ptr(idx),
                                           _ptr(shift), _ptr(M), _ptr(G), _ptr(B), _ptr(ws), ws.numel(),
                                           self._stream(stream)))
        return M, G, B

    def md_run(self, pos, vel, types, box, mass, dt, n_steps, rebuild_every, skin, capacity, stream=None):
        """mtp_md_run: velocity-Verlet on the device; pos / vel (torch CUDA, [N][3]) are updated in place.
        Returns dict(E[2] = potential, kinetic; Ei, F, virial, info[2])."""
        import torch
        n, dev = int(pos.shape[0]), pos.device
        wsb = C.c_size_t()
        self._check(_lib.mtp_md_workspace_bytes(self._h, n, int(capacity), C.byref(wsb)))
        ws = self._workspace(int(wsb.value), dev)
        out = dict(E=torch.empty(2, dtype=torch.float64, device=dev), Ei=torch.empty(n, dtype=torch.float64, device=dev),
                   F=torch.empty((n, 3), dtype=torch.float64, device=dev), virial=torch.empty(6, dtype=torch.float64, device=dev),
                   info=torch.zeros(2, dtype=torch.int64, device=dev))
        boxh = (C.c_double * 9)(*[float(x) for x in np.asarray(box, dtype=np.float64).reshape(9)])
        m = np.ascontiguousarray(mass, dtype=np.float64)
        self._check(_lib.mtp_md_run(self._h, n, _ptr(pos), _ptr(vel), _ptr(types), boxh, m.ctypes.data_as(C.POINTER(C.c_double)),
                                    float(dt), int(n_steps), int(rebuild_every), float(skin), int(capacity), _ptr(out["E"]),
                                    _ptr(out["Ei"]), _ptr(out["F"]), _ptr(out["virial"]), _ptr(out["info"]), _ptr(ws), ws.numel(),
                                    self._stream(stream)))
        return out

    def md_run_al(self, pos, vel, types, box, mass, dt, n_steps, rebuild_every, skin, capacity, Ainv, grade_every, mode,
                  select_threshold, break_threshold, max_selected, stream=None):
        """mtp_md_run_al: the MD loop with the grade policy.  Returns md_run's dict plus gamma_atom[N], selected
        [n_kept][N][3] (device), sel_step / sel_grade (lists), steps_done, n_evaluations, stopped, max_grade."""
        import torch
        n, dev = int(pos.shape[0]), pos.device
        wsb = C.c_size_t()
        self._check(_lib.mtp_md_al_workspace_bytes(self._h, n, int(capacity), C.byref(wsb)))
        ws = self._workspace(int(wsb.value), dev)
        out = dict(E=torch.empty(2, dtype=torch.float64, device=dev), Ei=torch.empty(n, dtype=torch.float64, device=dev),
                   F=torch.empty((n, 3), dtype=torch.float64, device=dev), virial=torch.empty(6, dtype=torch.float64, device=dev),
                   info=torch.zeros(2, dtype=torch.int64, device=dev), gamma_atom=torch.zeros(n, dtype=torch.float64, device=dev))
        sel = torch.empty((max(int(max_selected), 1), n, 3), dtype=torch.float64, device=dev)
        pol = AlPolicy(int(grade_every), int(mode), float(select_threshold), float(break_threshold), int(max_selected))
        sel_step = (C.c_int64 * max(int(max_selected), 1))()
        sel_grade = (C.c_double * max(int(max_selected), 1))()
        res = (C.c_int64 * 4)()
        mx = C.c_double()
        boxh = (C.c_double * 9)(*[float(x) for x in np.asarray(box, dtype=np.float64).reshape(9)])
        m = np.ascontiguousarray(mass, dtype=np.float64)
        self._check(_lib.mtp_md_run_al(self._h, n, _ptr(pos), _ptr(vel), _ptr(types), boxh, m.ctypes.data_as(C.POINTER(C.c_double)),
                                       float(dt), int(n_steps), int(rebuild_every), float(skin), int(capacity), _ptr(Ainv),
                                       C.byref(pol), _ptr(out["E"]), _ptr(out["Ei"]), _ptr(out["F"]), _ptr(out["virial"]),
                                       _ptr(out["info"]), _ptr(out["gamma_atom"]), _ptr(sel), sel_step, sel_grade, res, C.byref(mx),
                                       _ptr(ws), ws.numel(), self._stream(stream)))
        k = int(res[1])
        out.update(selected=sel[:k], sel_step=[int(sel_step[i]) for i in range(k)], sel_grade=[float(sel_grade[i]) for i in range(k)],
                   steps_done=int(res[0]), n_evaluations=int(res[2]), stopped=bool(res[3]), max_grade=float(mx.value))
        return out

    def compute_host_pos(self, pos, types, box, out=None):
        """mtp_compute_host_pos on numpy (or pinned) arrays: positions in, forces out, list built on the device."""
        n = int(pos.shape[0])
        if out is None:
            out = dict(E=np.empty(1), Ei=np.empty(n), F=np.empty((n, 3)), virial=np.empty(6))
        boxh = (C.c_double * 9)(*[float(x) for x in np.asarray(box, dtype=np.float64).reshape(9)])
        nnz = C.c_int64()
        self._check(_lib.mtp_compute_host_pos(self._h, n, _np_ptr(pos), _np_ptr(types), boxh, _np_ptr(out["E"]), _np_ptr(out["Ei"]),
                                              _np_ptr(out["F"]), _np_ptr(out["virial"]), C.byref(nnz)))
        out["nnz"] = int(nnz.value)
        return out

    def compute_host(self, pos, types, box, off, idx, shift=None, rev=None, out=None):
        """mtp_compute_host on numpy (or pinned torch CPU) arrays; H2D/D2H inside the call."""
        n, nnz = int(pos.shape[0]), int(idx.shape[0])
        if out is None:
            out = dict(E=np.empty(1), Ei=np.empty(n), F=np.empty((n, 3)), virial=np.empty(6))
        boxh = (C.c_double * 9)(*[float(x) for x in np.asarray(box, dtype=np.float64).reshape(9)])
        self._check(_lib.mtp_compute_host(self._h, n, _np_ptr(pos), _np_ptr(types), boxh, _np_ptr(off), _np_ptr(idx),
                                          _np_ptr(shift), _np_ptr(rev), nnz, _np_ptr(out["E"]), _np_ptr(out["Ei"]),
                                          _np_ptr(out["F"]), _np_ptr(out["virial"])))
        return out


def dump_selected(path, run, types, box, append=True):
    """The dump step of the grade policy ("the current configuration is written to the output file"): the
    configurations md_run_al kept, as extended-XYZ text frames (species index, x, y, z per atom; lattice, step and
    grade in the comment line).  The MLIP-3 .cfg format of the paper is not reproduced (its specification is not
    available here).  Returns the number of frames written."""
    box = np.asarray(box, dtype=np.float64).reshape(9)
    types = np.asarray(types.cpu() if hasattr(types, "cpu") else types)
    sel = run["selected"].cpu().numpy() if hasattr(run["selected"], "cpu") else np.asarray(run["selected"])
    with open(path, "a" if append else "w") as f:
        for k, (step, grade) in enumerate(zip(run["sel_step"], run["sel_grade"])):
            f.write("%d\n" % sel.shape[1])
            f.write('Lattice="%s" Properties=species:I:1:pos:R:3 step=%d grade=%.17g\n' % (" ".join("%.17g" % v for v in box), step, grade))
            for t, (x, y, z) in zip(types, sel[k]):
                f.write("%d %.17g %.17g %.17g\n" % (int(t), x, y, z))
    return len(run["sel_step"])


class ComputeGraph:
    """An mtp_graph: one captured mtp_compute call."""

    def __init__(self, pot, g, keep):
        self._pot, self._g, self._keep = pot, g, keep

    def launch(self, stream=None):
        rc = _lib.mtp_graph_launch(self._g, Potential._stream(stream))
        if rc != OK:
            raise MtpError(rc, "mtp_graph_launch")

    def close(self):
        if self._g:
            _lib.mtp_graph_destroy(self._g)
            self._g = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def neighbors_build(pos, box, r_list, capacity=None, want_rev=True, stream=None):
    """mtp_neighbors_build on a torch CUDA tensor pos [N][3].  capacity None: count first, then build exactly.
    Returns dict(off, idx, shift, rev, nnz, errors); tensors are sized `capacity` (nnz of them valid)."""
    import torch
    n, dev = int(pos.shape[0]), pos.device
    wsb = C.c_size_t()
    rc = _lib.mtp_neighbors_workspace_bytes(n, C.byref(wsb))
    if rc != OK:
        raise MtpError(rc, "mtp_neighbors_workspace_bytes")
    ws = torch.empty(int(wsb.value), dtype=torch.uint8, device=dev)
    boxh = (C.c_double * 9)(*[float(x) for x in np.asarray(box, dtype=np.float64).reshape(9)])
    off = torch.empty(n + 1, dtype=torch.int64, device=dev)
    info = torch.zeros(2, dtype=torch.int64, device=dev)
    st = Potential._stream(stream)

    def run(cap):
        idx = torch.empty(max(cap, 1), dtype=torch.int32, device=dev)
        shift = torch.empty((max(cap, 1), 3), dtype=torch.int8, device=dev)
        rev = torch.empty(max(cap, 1), dtype=torch.int32, device=dev) if want_rev else None
        rc = _lib.mtp_neighbors_build(n, _ptr(pos), boxh, float(r_list), int(cap), _ptr(off), _ptr(idx), _ptr(shift), _ptr(rev),
                                      _ptr(info), _ptr(ws), ws.numel(), st)
        if rc != OK:
            raise MtpError(rc, "mtp_neighbors_build")
        return idx, shift, rev

    if capacity is None:
        run(0)
        capacity = int(info.cpu()[0])
    idx, shift, rev = run(int(capacity))
    nnz, errors = [int(x) for x in info.cpu()]
    return dict(off=off, idx=idx, shift=shift, rev=rev, nnz=nnz, errors=errors)


NB_STATIC_MAX_ATOMS = 32768


def neighbors_build_static(pos, box, r_list, off, idx, shift, rev, info, stream=None):
    """mtp_neighbors_build_static: the list build with no workspace argument and no allocation (limit
    NB_STATIC_MAX_ATOMS atoms).  Every output is the caller's torch CUDA tensor: off [N+1] i64, idx [cap] i32,
    shift [cap][3] i8, rev [cap] i32 or None, info [2] i64 (pairs found, errors).  Nothing is read back or
    synchronised here."""
    n, cap = int(pos.shape[0]), int(idx.shape[0])
    boxh = (C.c_double * 9)(*[float(x) for x in np.asarray(box, dtype=np.float64).reshape(9)])
    rc = _lib.mtp_neighbors_build_static(n, _ptr(pos), boxh, float(r_list), cap, _ptr(off), _ptr(idx), _ptr(shift), _ptr(rev),
                                         _ptr(info), Potential._stream(stream))
    if rc != OK:
        raise MtpError(rc, "mtp_neighbors_build_static: " + _lib.mtp_last_error(None).decode())
    return rc


def launch_count() -> int:
    return int(_lib.mtp_launch_count())


def peak_dfma(iters: int, sink, stream=None):
    """Enqueue the fp64-FMA microbenchmark; returns the flop count of the launch."""
    fl = C.c_double()
    rc = _lib.mtp_peak_dfma(int(iters), _ptr(sink), C.byref(fl), Potential._stream(stream))
    if rc != OK:
        raise MtpError(rc, "mtp_peak_dfma")
    return fl.value
