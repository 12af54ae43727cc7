"""ctypes front end of the CPU oracle (oracle/csf_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module. It shares no code with the CUDA
path; both are driven with the same seeded inputs from paper_2410_02754_b200.synth.

All arrays are host NumPy arrays. A spinor block is complex128 of shape [2M, nvec] (row 2I+alpha,
vector fastest).
"""
import ctypes as C
import numpy as np

from . import build as _build

_lib = None

BC_PERIODIC, BC_DIRICHLET, BC_FREE = 0, 1, 2


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.ref_num_threads.restype = C.c_int
    return _lib


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t))


def _chk(rc, what):
    if rc != 0:
        raise RuntimeError(f"oracle {what} failed with code {rc}")


def gll(p):
    x = np.zeros(p + 1); w = np.zeros(p + 1)
    _chk(lib().ref_gll(C.c_int(p), _p(x, C.c_double), _p(w, C.c_double)), "gll")
    return x, w


def gauss_legendre(nq):
    x = np.zeros(nq); w = np.zeros(nq)
    _chk(lib().ref_gauss_legendre(C.c_int(nq), _p(x, C.c_double), _p(w, C.c_double)), "gauss_legendre")
    return x, w


def ref1d(p):
    n = p + 1
    K = np.zeros((n, n)); M = np.zeros((n, n)); D = np.zeros((n, n))
    _chk(lib().ref_ref1d(C.c_int(p), _p(K, C.c_double), _p(M, C.c_double), _p(D, C.c_double)), "ref1d")
    return K, M, D


def num_threads():
    return int(lib().ref_num_threads())


class RefCtx:
    """Oracle context: mesh, lumped mass, sparse-assembled 1/2 K, nodal potential, projectors."""

    def __init__(self, ncell, box, order, bc, assemble_sparse=True):
        self._h = C.c_void_p()
        nc = (C.c_int * 3)(*[int(v) for v in ncell]); bx = (C.c_double * 3)(*[float(v) for v in box])
        b = (C.c_int * 3)(*[int(v) for v in bc])
        _chk(lib().ref_create2(C.byref(self._h), nc, bx, C.c_int(order), b, C.c_int(1 if assemble_sparse else 0)), "create")
        self.ncell = tuple(int(v) for v in ncell); self.box = tuple(float(v) for v in box)
        self.order = int(order); self.bc = tuple(int(v) for v in bc)
        m = C.c_int64(); _chk(lib().ref_num_nodes(self._h, C.byref(m)), "num_nodes"); self.M = int(m.value)
        e = C.c_int64(); _chk(lib().ref_num_cells(self._h, C.byref(e)), "num_cells"); self.E = int(e.value)

    def close(self):
        if self._h:
            lib().ref_destroy(self._h); self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def node_coords(self):
        xyz = np.zeros((self.M, 3)); _chk(lib().ref_node_coords(self._h, _p(xyz, C.c_double)), "node_coords"); return xyz

    def mass_diag(self):
        m = np.zeros(self.M); _chk(lib().ref_mass_diag(self._h, _p(m, C.c_double)), "mass_diag"); return m

    def connectivity(self):
        n3 = (self.order + 1) ** 3
        conn = np.zeros((self.E, n3), dtype=np.int64); _chk(lib().ref_connectivity(self._h, _p(conn, C.c_int64)), "connectivity"); return conn

    def cell_matrix(self):
        n3 = (self.order + 1) ** 3
        Ke = np.zeros((n3, n3)); _chk(lib().ref_cell_matrix(self._h, _p(Ke, C.c_double)), "cell_matrix"); return Ke

    def csr(self):
        """(rowptr, col, val) of the assembled real M x M matrix 1/2 K."""
        nnz = C.c_int64(); _chk(lib().ref_csr_nnz(self._h, C.byref(nnz)), "csr_nnz")
        rowptr = np.zeros(self.M + 1, dtype=np.int64); col = np.zeros(nnz.value, dtype=np.int32); val = np.zeros(nnz.value)
        _chk(lib().ref_csr(self._h, _p(rowptr, C.c_int64), _p(col, C.c_int32), _p(val, C.c_double)), "csr")
        return rowptr, col, val

    def set_potential(self, veff, bxyz=None):
        veff = np.ascontiguousarray(veff, dtype=np.float64); assert veff.shape == (self.M,)
        if bxyz is not None:
            bxyz = np.ascontiguousarray(bxyz, dtype=np.float64); assert bxyz.shape == (self.M, 3)
        _chk(lib().ref_set_potential(self._h, _p(veff, C.c_double), _p(bxyz, C.c_double) if bxyz is not None else None), "set_potential")

    def set_projectors(self, node_ptr, node_idx, nproj, pvals, atom_type, delta, delta_ptr):
        natoms = len(nproj)
        if natoms == 0:
            _chk(lib().ref_set_projectors(self._h, C.c_int(0), None, None, None, None, None, C.c_int(0), None, None), "set_projectors"); return
        node_ptr = np.ascontiguousarray(node_ptr, dtype=np.int64); node_idx = np.ascontiguousarray(node_idx, dtype=np.int64)
        nproj = np.ascontiguousarray(nproj, dtype=np.int32); pvals = np.ascontiguousarray(pvals, dtype=np.float64)
        atom_type = np.ascontiguousarray(atom_type, dtype=np.int32)
        delta = np.ascontiguousarray(delta, dtype=np.complex128); delta_ptr = np.ascontiguousarray(delta_ptr, dtype=np.int64)
        _chk(lib().ref_set_projectors(self._h, C.c_int(natoms), _p(node_ptr, C.c_int64), _p(node_idx, C.c_int64), _p(nproj, C.c_int),
                                      _p(pvals, C.c_double), _p(atom_type, C.c_int), C.c_int(len(delta_ptr) - 1),
                                      delta.ctypes.data_as(C.c_void_p), _p(delta_ptr, C.c_int64)), "set_projectors")

    def _xy(self, X):
        X = np.ascontiguousarray(X, dtype=np.complex128); assert X.ndim == 2 and X.shape[0] == 2 * self.M
        return X, np.zeros_like(X)

    def apply_H(self, X):
        X, Y = self._xy(X); nv = X.shape[1]
        _chk(lib().ref_apply_H(self._h, X.ctypes.data_as(C.c_void_p), Y.ctypes.data_as(C.c_void_p), C.c_int64(nv), C.c_int(nv)), "apply_H")
        return Y

    def apply_H_rows(self, X, rows):
        X = np.ascontiguousarray(X, dtype=np.complex128); rows = np.ascontiguousarray(rows, dtype=np.int64); nv = X.shape[1]
        out = np.zeros((len(rows), nv), dtype=np.complex128)
        _chk(lib().ref_apply_H_rows(self._h, X.ctypes.data_as(C.c_void_p), C.c_int64(nv), C.c_int(nv), _p(rows, C.c_int64), C.c_int(len(rows)),
                                    out.ctypes.data_as(C.c_void_p)), "apply_H_rows")
        return out

    def filter(self, X, degree, a, b):
        X, Y = self._xy(X); nv = X.shape[1]
        _chk(lib().ref_filter(self._h, X.ctypes.data_as(C.c_void_p), Y.ctypes.data_as(C.c_void_p), C.c_int64(nv), C.c_int(nv),
                              C.c_int(degree), C.c_double(a), C.c_double(b)), "filter")
        return Y

    def dense_H(self):
        """O9: Hhat as a dense (2M x 2M) array = apply_H on the identity (tiny meshes only)."""
        return self.apply_H(np.eye(2 * self.M, dtype=np.complex128))
