"""Thin Python binding of libcsf.so (include/csf.h): argument marshalling only.

Every step of the path runs in the library's CUDA kernels; PyTorch is used for device memory and streams.
There is no CPU fallback: if libcsf.so is missing or no CUDA device is present, calls raise.
"""
import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libcsf.so")

CSF_OK, CSF_EINVAL, CSF_ENOMEM, CSF_ECUDA, CSF_ESTATE, CSF_EUNSUPPORTED = 0, -1, -2, -3, -4, -5
CSF_BC_PERIODIC, CSF_BC_DIRICHLET, CSF_BC_FREE = 0, 1, 2
CSF_FP64, CSF_FP32_INTERMEDIATE = 0, 1
STATIC_SCRATCH_BYTES = 8 << 20          # CSF_STATIC_SCRATCH_BYTES of include/csf.h

EXPORTS = ["csf_create", "csf_destroy", "csf_set_stream", "csf_num_nodes", "csf_node_coords", "csf_mass_diag", "csf_set_potential",
           "csf_set_projectors", "csf_workspace_bytes", "csf_apply_H", "csf_apply_H_static", "csf_filter", "csf_filter_host", "csf_set_host_chunk",
           "csf_profile_enable", "csf_profile_read", "csf_probe_fp64_peak", "csf_probe_fp64_mixed", "csf_launch_count", "csf_column_lanes", "csf_filter_fused_gather", "csf_set_variant", "csf_set_tuning", "csf_last_error",
           "csf_rr_workspace_bytes", "csf_rr_project", "csf_rr_solve", "csf_rr_rotate", "csf_density", "csf_lanczos_workspace_bytes", "csf_lanczos",
           "csf_tridiag_extremes", "csf_quadrature_points", "csf_set_potential_quadrature", "csf_dense_workspace_bytes", "csf_apply_H_dense",
           "csf_filter_dense", "csf_set_kpoint", "csf_set_projectors_complex"]
KIND_CELL, KIND_PGATHER, KIND_DELTA, KIND_AUX = 0, 1, 2, 3
KIND_NAMES = ("cell", "proj_gather", "delta", "aux")

_lib = None


class CsfError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libcsf error {code}: {msg}")
        self.code = code


def lib():
    """Load libcsf.so (built in-tree by paper_2410_02754_b200/build.py). Fails loudly if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise FileNotFoundError(f"{LIB_PATH} not found: run `python -m paper_2410_02754_b200.build` (no CPU fallback exists)")
        _lib = C.CDLL(LIB_PATH)
        _lib.csf_last_error.restype = C.c_char_p
        _lib.csf_last_error.argtypes = [C.c_void_p]
    return _lib


def _dp(a, t):
    return a.ctypes.data_as(C.POINTER(t))


class Csf:
    """One mesh + operator context on one GPU. Method names mirror the C entry points."""

    def __init__(self, ncell, box, order, bc, device=0, stream=None):
        self._h = C.c_void_p()
        self._L = lib()
        nc = (C.c_int * 3)(*[int(v) for v in ncell]); bx = (C.c_double * 3)(*[float(v) for v in box]); b = (C.c_int * 3)(*[int(v) for v in bc])
        rc = self._L.csf_create(C.byref(self._h), nc, bx, C.c_int(int(order)), b, C.c_int(int(device)), C.c_void_p(stream or 0))
        if rc != CSF_OK:
            raise CsfError(rc, self._L.csf_last_error(None).decode())
        self.ncell, self.box, self.order, self.bc, self.device = tuple(ncell), tuple(box), int(order), tuple(bc), int(device)
        m = C.c_int64(); self._chk(self._L.csf_num_nodes(self._h, C.byref(m))); self.M = int(m.value)
        self.E = int(self.ncell[0]) * int(self.ncell[1]) * int(self.ncell[2])

    def _chk(self, rc):
        if rc != CSF_OK:
            raise CsfError(rc, self._L.csf_last_error(self._h).decode())

    def destroy(self):
        if self._h:
            self._L.csf_destroy(self._h); self._h = C.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def set_stream(self, stream):
        self._chk(self._L.csf_set_stream(self._h, C.c_void_p(stream or 0)))

    def node_coords(self):
        xyz = np.zeros((self.M, 3)); self._chk(self._L.csf_node_coords(self._h, _dp(xyz, C.c_double))); return xyz

    def mass_diag(self):
        m = np.zeros(self.M); self._chk(self._L.csf_mass_diag(self._h, _dp(m, C.c_double))); return m

    def set_potential(self, veff, bxyz=None):
        veff = np.ascontiguousarray(veff, dtype=np.float64)
        if veff.shape != (self.M,):
            raise ValueError("veff must have shape [M]")
        if bxyz is not None:
            bxyz = np.ascontiguousarray(bxyz, dtype=np.float64)
            if bxyz.shape != (self.M, 3):
                raise ValueError("bxyz must have shape [M,3]")
        self._chk(self._L.csf_set_potential(self._h, _dp(veff, C.c_double), _dp(bxyz, C.c_double) if bxyz is not None else None))

    def set_projectors(self, node_ptr, node_idx, nproj, pvals, atom_type, delta, delta_ptr):
        natoms = len(nproj)
        if natoms == 0:
            self._chk(self._L.csf_set_projectors(self._h, C.c_int(0), None, None, None, None, None, C.c_int(0), None, None)); return
        node_ptr = np.ascontiguousarray(node_ptr, dtype=np.int64); node_idx = np.ascontiguousarray(node_idx, dtype=np.int64)
        nproj = np.ascontiguousarray(nproj, dtype=np.int32); pvals = np.ascontiguousarray(pvals, dtype=np.float64)
        atom_type = np.ascontiguousarray(atom_type, dtype=np.int32)
        delta = np.ascontiguousarray(delta, dtype=np.complex128); delta_ptr = np.ascontiguousarray(delta_ptr, dtype=np.int64)
        self._chk(self._L.csf_set_projectors(self._h, C.c_int(natoms), _dp(node_ptr, C.c_int64), _dp(node_idx, C.c_int64), _dp(nproj, C.c_int),
                                             _dp(pvals, C.c_double), _dp(atom_type, C.c_int), C.c_int(len(delta_ptr) - 1),
                                             delta.ctypes.data_as(C.c_void_p), _dp(delta_ptr, C.c_int64)))

    def set_projectors_complex(self, node_ptr, node_idx, nproj, pvals, atom_type, delta, delta_ptr):
        """set_projectors with complex entries P^{a,k}_{I chi} (eq.42); served by the dense path only."""
        natoms = len(nproj)
        if natoms == 0:
            self._chk(self._L.csf_set_projectors_complex(self._h, C.c_int(0), None, None, None, None, None, C.c_int(0), None, None)); return
        node_ptr = np.ascontiguousarray(node_ptr, dtype=np.int64); node_idx = np.ascontiguousarray(node_idx, dtype=np.int64)
        nproj = np.ascontiguousarray(nproj, dtype=np.int32); pvals = np.ascontiguousarray(pvals, dtype=np.complex128)
        atom_type = np.ascontiguousarray(atom_type, dtype=np.int32)
        delta = np.ascontiguousarray(delta, dtype=np.complex128); delta_ptr = np.ascontiguousarray(delta_ptr, dtype=np.int64)
        self._chk(self._L.csf_set_projectors_complex(self._h, C.c_int(natoms), _dp(node_ptr, C.c_int64), _dp(node_idx, C.c_int64), _dp(nproj, C.c_int),
                                                     pvals.ctypes.data_as(C.c_void_p), _dp(atom_type, C.c_int), C.c_int(len(delta_ptr) - 1),
                                                     delta.ctypes.data_as(C.c_void_p), _dp(delta_ptr, C.c_int64)))

    def set_kpoint(self, kvec):
        """Bloch vector (1/bohr); call set_potential_quadrature after it."""
        k = np.ascontiguousarray(kvec, dtype=np.float64); assert k.shape == (3,)
        self._chk(self._L.csf_set_kpoint(self._h, _dp(k, C.c_double)))

    def workspace_bytes(self, nvec, mode=CSF_FP64):
        b = C.c_size_t(); self._chk(self._L.csf_workspace_bytes(self._h, C.c_int(int(nvec)), C.c_int(mode), C.byref(b))); return int(b.value)

    # ---- device entry points: raw pointers (ints) or torch tensors ----
    @staticmethod
    def _ptr(t):
        return C.c_void_p(t if isinstance(t, int) else t.data_ptr())

    @staticmethod
    def _nbytes(t, given):
        return C.c_size_t(given if isinstance(t, int) else t.numel() * t.element_size())

    def apply_H(self, dX, dY, ld, nvec, d_work, work_bytes=0):
        self._chk(self._L.csf_apply_H(self._h, self._ptr(dX), self._ptr(dY), C.c_int64(int(ld)), C.c_int(int(nvec)), self._ptr(d_work), self._nbytes(d_work, work_bytes)))

    def apply_H_static(self, dX, dY, ld, nvec):
        """csf_apply_H without a workspace and without any allocation: the scratch is a static array inside the library
        (STATIC_SCRATCH_BYTES); calls on one device share it and must not overlap on the GPU."""
        self._chk(self._L.csf_apply_H_static(self._h, self._ptr(dX), self._ptr(dY), C.c_int64(int(ld)), C.c_int(int(nvec))))

    # ---- general quadrature rule, dense cell-matrix apply
    def quadrature_points(self, nq):
        """[E, nq^3, 3] coordinates of the Gauss-Legendre points of every cell."""
        out = np.empty((self.E, int(nq) ** 3, 3), dtype=np.float64)
        self._chk(self._L.csf_quadrature_points(self._h, C.c_int(int(nq)), _dp(out, C.c_double)))
        return out

    def set_potential_quadrature(self, nq, vq):
        """vq[E, nq^3, 4] = V_eff, B_x, B_y, B_z at the quadrature points."""
        vq = np.ascontiguousarray(vq, dtype=np.float64)
        assert vq.shape == (self.E, int(nq) ** 3, 4), "vq must be [E, nq^3, 4]"
        self._chk(self._L.csf_set_potential_quadrature(self._h, C.c_int(int(nq)), _dp(vq, C.c_double)))

    def dense_workspace_bytes(self, nvec):
        b = C.c_size_t()
        self._chk(self._L.csf_dense_workspace_bytes(self._h, C.c_int(int(nvec)), C.byref(b)))
        return int(b.value)

    def apply_H_dense(self, dX, dY, ld, nvec, d_work=0, work_bytes=0):
        self._chk(self._L.csf_apply_H_dense(self._h, self._ptr(dX), self._ptr(dY), C.c_int64(int(ld)), C.c_int(int(nvec)), self._ptr(d_work), self._nbytes(d_work, work_bytes)))

    def filter_dense(self, dX, dY, ld, nvec, degree, a, b, d_work=0, work_bytes=0):
        self._chk(self._L.csf_filter_dense(self._h, self._ptr(dX), self._ptr(dY), C.c_int64(int(ld)), C.c_int(int(nvec)), C.c_int(int(degree)),
                                           C.c_double(float(a)), C.c_double(float(b)), self._ptr(d_work), self._nbytes(d_work, work_bytes)))

    def filter(self, dX, dY, ld, nvec, degree, a, b, mode=CSF_FP64, d_work=0, work_bytes=0):
        self._chk(self._L.csf_filter(self._h, self._ptr(dX), self._ptr(dY), C.c_int64(int(ld)), C.c_int(int(nvec)), C.c_int(int(degree)),
                                     C.c_double(float(a)), C.c_double(float(b)), C.c_int(mode), self._ptr(d_work), self._nbytes(d_work, work_bytes)))

    def filter_host(self, hX, hY, ld, nvec, degree, a, b, mode=CSF_FP64):
        """hX, hY: host pointers (ints), NumPy arrays or CPU (pinned) torch tensors."""
        def hp(t):
            if isinstance(t, int):
                return C.c_void_p(t)
            if isinstance(t, np.ndarray):
                return C.c_void_p(t.ctypes.data)
            return C.c_void_p(t.data_ptr())
        self._chk(self._L.csf_filter_host(self._h, hp(hX), hp(hY), C.c_int64(int(ld)), C.c_int(int(nvec)), C.c_int(int(degree)),
                                          C.c_double(float(a)), C.c_double(float(b)), C.c_int(mode)))

    def set_host_chunk(self, ncols):
        self._chk(self._L.csf_set_host_chunk(self._h, C.c_int(int(ncols))))

    def profile_enable(self, on=True):
        self._chk(self._L.csf_profile_enable(self._h, C.c_int(1 if on else 0)))

    def profile_read(self, kind):
        """(summed device ms, launches) of kernel kind since the last read; synchronises the stream."""
        ms = C.c_double(); n = C.c_int64()
        self._chk(self._L.csf_profile_read(self._h, C.c_int(int(kind)), C.byref(ms), C.byref(n)))
        return float(ms.value), int(n.value)

    def column_lanes(self, nvec, mode=0):
        n = C.c_int(); self._chk(self._L.csf_column_lanes(self._h, C.c_int(int(nvec)), C.c_int(int(mode)), C.byref(n))); return int(n.value)

    def filter_fused_gather(self, nvec, mode=0):
        n = C.c_int(); self._chk(self._L.csf_filter_fused_gather(self._h, C.c_int(int(nvec)), C.c_int(int(mode)), C.byref(n))); return bool(n.value)

    def launch_count(self):
        n = C.c_int64(); self._chk(self._L.csf_launch_count(self._h, C.byref(n))); return int(n.value)

    # ---- subspace steps
    def rr_workspace_bytes(self, nvec):
        b = C.c_size_t(); self._chk(self._L.csf_rr_workspace_bytes(self._h, C.c_int(int(nvec)), C.byref(b))); return int(b.value)

    def rr_project(self, dX, ld, nvec, dHs, dSs, d_work, work_bytes=0):
        self._chk(self._L.csf_rr_project(self._h, self._ptr(dX), C.c_int64(int(ld)), C.c_int(int(nvec)), self._ptr(dHs), self._ptr(dSs), self._ptr(d_work), self._nbytes(d_work, work_bytes)))

    def rr_solve(self, dHs, dSs, n, dQ):
        """Returns the Ritz values (host NumPy array, ascending); dQ receives the eigenvectors on the device."""
        lam = np.zeros(int(n))
        self._chk(self._L.csf_rr_solve(self._h, self._ptr(dHs), self._ptr(dSs), C.c_int(int(n)), self._ptr(dQ), _dp(lam, C.c_double)))
        return lam

    def rr_rotate(self, dX, ld, nvec, dQ, dU, ldu, d_work, work_bytes=0):
        self._chk(self._L.csf_rr_rotate(self._h, self._ptr(dX), C.c_int64(int(ld)), C.c_int(int(nvec)), self._ptr(dQ), self._ptr(dU), C.c_int64(int(ldu)), self._ptr(d_work), self._nbytes(d_work, work_bytes)))

    def density(self, dX, ld, nvec, occ, d_rho_m, accumulate=False):
        occ = np.ascontiguousarray(occ, dtype=np.float64)
        if occ.shape != (int(nvec),):
            raise ValueError("occ must have shape [nvec]")
        self._chk(self._L.csf_density(self._h, self._ptr(dX), C.c_int64(int(ld)), C.c_int(int(nvec)), _dp(occ, C.c_double), self._ptr(d_rho_m), C.c_int(1 if accumulate else 0)))

    def lanczos_workspace_bytes(self):
        b = C.c_size_t(); self._chk(self._L.csf_lanczos_workspace_bytes(self._h, C.byref(b))); return int(b.value)

    def lanczos(self, d_v0, k, d_work, work_bytes=0):
        """(alpha, beta) of k Lanczos steps on Hhat from the device vector d_v0 (host NumPy arrays, truncated to the steps taken)."""
        al = np.zeros(int(k)); be = np.zeros(int(k)); done = C.c_int()
        self._chk(self._L.csf_lanczos(self._h, self._ptr(d_v0), C.c_int(int(k)), _dp(al, C.c_double), _dp(be, C.c_double), C.byref(done), self._ptr(d_work), self._nbytes(d_work, work_bytes)))
        return al[:done.value], be[:done.value]

    def set_tuning(self, seg_len=0, chunk_group=16):
        self._chk(self._L.csf_set_tuning(self._h, C.c_int(int(seg_len)), C.c_int(int(chunk_group))))

    def set_variant(self, variant):
        self._chk(self._L.csf_set_variant(self._h, C.c_int(int(variant))))


def probe_fp64_mixed(device=0):
    """TFLOP/s of DFMA and DMMA loops running side by side on every SM (csf_probe_fp64_mixed)."""
    t = C.c_double()
    rc = lib().csf_probe_fp64_mixed(C.c_int(int(device)), C.byref(t))
    if rc != CSF_OK:
        raise CsfError(rc, lib().csf_last_error(None).decode())
    return float(t.value)


def tridiag_extremes(alpha, beta):
    """(theta_min, theta_max) of the Lanczos tridiagonal matrix (csf_tridiag_extremes: Sturm bisection in the library)."""
    alpha = np.ascontiguousarray(alpha, dtype=np.float64); beta = np.ascontiguousarray(beta, dtype=np.float64)
    lo = C.c_double(); hi = C.c_double()
    rc = lib().csf_tridiag_extremes(_dp(alpha, C.c_double), _dp(beta, C.c_double), C.c_int(len(alpha)), C.byref(lo), C.byref(hi))
    if rc != CSF_OK:
        raise CsfError(rc, "csf_tridiag_extremes")
    return float(lo.value), float(hi.value)


def probe_fp64_peak(device=0):
    """(TFLOP/s of a register-resident DFMA loop, TFLOP/s of a DMMA m8n8k4 loop) measured on `device`."""
    f = C.c_double(); m = C.c_double()
    rc = lib().csf_probe_fp64_peak(C.c_int(int(device)), C.byref(f), C.byref(m))
    if rc != CSF_OK:
        raise CsfError(rc, lib().csf_last_error(None).decode())
    return float(f.value), float(m.value)
