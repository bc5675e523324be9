"""Thin ctypes binding of libhprmat.so (include/hprmat.h): argument marshalling only, same names as the C ABI.

Device buffers are torch CUDA tensors (PyTorch is used for device memory and streams only); every arithmetic step
runs in the library's own sm_100a kernels.  There is no CPU fallback: if the shared library is missing or no CUDA
device is present the calls raise.
"""
import ctypes as C
import os

import numpy as np
import torch

HERE = os.path.dirname(os.path.abspath(__file__))
LIBPATH = os.path.join(HERE, "libhprmat.so")

HPRMAT_FP64, HPRMAT_MIXED, HPRMAT_MIXED_REFINE, HPRMAT_TYPE3 = 1, 2, 3, 4
HPRMAT_OK, HPRMAT_ESINGULAR, HPRMAT_ENOTCONVERGED, HPRMAT_ENOMEM, HPRMAT_ECUDA, HPRMAT_EUNVERIFIED = 0, 1, 2, 3, 4, 5
HPRMAT_OPT_FP64_ALGO, HPRMAT_OPT_ZGEMM_ALGO, HPRMAT_OPT_GRAPHS = 1, 2, 3
MODES = {"fp64": HPRMAT_FP64, "mixed": HPRMAT_MIXED, "mixed_refine": HPRMAT_MIXED_REFINE, "type3": HPRMAT_TYPE3}


class hprmat_info(C.Structure):
    _fields_ = [("status", C.c_int), ("refine_steps", C.c_int), ("pivot_index", C.c_int), ("reserved", C.c_int),
                ("resid_max", C.c_double), ("backward_err", C.c_double),
                ("ms_assemble", C.c_double), ("ms_lu", C.c_double), ("ms_solve", C.c_double),
                ("ms_refine", C.c_double), ("ms_contract", C.c_double), ("ms_total", C.c_double),
                ("lu_tflops", C.c_double)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


class HprmatError(RuntimeError):
    def __init__(self, code, where):
        self.code = code
        msg = lib().hprmat_strerror(C.c_int(code)).decode()
        if code == HPRMAT_ECUDA:
            msg += ": " + lib().hprmat_last_cuda_error().decode()
        super().__init__(f"{where}: rc={code} ({msg})")


_lib = None


def lib():
    """Load libhprmat.so (built in-tree by paper_2512_11590_b200.build); fails loudly if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIBPATH):
            raise ImportError(f"{LIBPATH} not found: run `python -m paper_2512_11590_b200.build` (no CPU fallback)")
        L = C.CDLL(LIBPATH)
        L.hprmat_strerror.restype = C.c_char_p
        L.hprmat_last_cuda_error.restype = C.c_char_p
        L.hprmat_launch_count.restype = C.c_longlong
        L.hprmat_workspace_bytes.restype = C.c_size_t
        L.hprmat_collision_workspace_bytes.restype = C.c_size_t
        L.hprmat_propagate_workspace_bytes.restype = C.c_size_t
        _lib = L
    return _lib


def _dev(t: torch.Tensor):
    assert t.is_cuda, "device pointer expected"
    return C.c_void_p(t.data_ptr())


def _stream(stream=None):
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def _check(rc, where, ok=(HPRMAT_OK,)):
    if rc not in ok:
        raise HprmatError(rc, where)
    return rc


def hprmat_launch_count() -> int:
    return int(lib().hprmat_launch_count())


def hprmat_profile(enable: bool):
    _check(lib().hprmat_profile(C.c_int(1 if enable else 0)), "hprmat_profile")


def hprmat_profile_read():
    ms, fl, n = C.c_double(0), C.c_double(0), C.c_longlong(0)
    _check(lib().hprmat_profile_read(C.byref(ms), C.byref(fl), C.byref(n)), "hprmat_profile_read")
    return ms.value, fl.value, n.value


def hprmat_profile_cgemm_variant(variant: int = -1) -> int:
    """Select (0 auto, 1 one-tile-per-CTA, 2 persistent, 3 / 4 persistent CTA pairs with 256 x 128 / 256 x 256 tiles) or query the complex64 GEMM kernel."""
    return int(lib().hprmat_profile_cgemm_variant(C.c_int(variant)))


def hprmat_profile_cgemm3_variant(variant: int) -> int:
    """0 auto, 1 mma.sync, 2 tcgen05 (operand split in shared memory) for the FP32-class complex64 GEMM."""
    return int(lib().hprmat_profile_cgemm3_variant(C.c_int(variant)))


def hprmat_profile_pdl(enable: int = -1) -> int:
    """Programmatic dependent launch of the small LU kernels: 1 on (default), 0 off, anything else queries."""
    return int(lib().hprmat_profile_pdl(C.c_int(enable)))


def hprmat_profile_lookahead(enable: int = -1) -> int:
    """Look-ahead inside the verified-diagonal factorisations: 1 on (default), 0 off, anything else queries."""
    return int(lib().hprmat_profile_lookahead(C.c_int(enable)))


PROF_CATS = ("lu_gemm", "lu_trsm", "panel", "laswp", "solve", "other")


def hprmat_profile_cat(cat: int):
    ms, fl, n = C.c_double(0), C.c_double(0), C.c_longlong(0)
    _check(lib().hprmat_profile_cat(C.c_int(cat), C.byref(ms), C.byref(fl), C.byref(n)), "hprmat_profile_cat")
    return ms.value, fl.value, n.value


_bench_lib = None


def hprmat_bench_dmma_peak(iters=20000, ctas_per_sm=2, stream=None):
    """FP64 tensor-core issue-rate ceiling (TFLOP/s, ms) from libhprmat_bench.so -- bench.py's roofline denominator; the
    product library does not contain this probe (include/hprmat_profile.h)."""
    global _bench_lib
    if _bench_lib is None:
        path = os.path.join(HERE, "libhprmat_bench.so")
        if not os.path.exists(path):
            raise ImportError(f"{path} not found: run `python -m paper_2512_11590_b200.build`")
        _bench_lib = C.CDLL(path)
    tf, ms = C.c_double(0), C.c_double(0)
    _check(_bench_lib.hprmat_bench_dmma_peak(_stream(stream), C.c_int(iters), C.c_int(ctas_per_sm), C.byref(tf), C.byref(ms)),
           "hprmat_bench_dmma_peak")
    return tf.value, ms.value


# ---- structured R-matrix path ---------------------------------------------------------------------------------------
class Context:
    """Owner of an hprmat_ctx (hprmat_setup ... hprmat_destroy)."""

    def __init__(self, nch, nbasis, a, h2m, lval, ethr, max_mode=0, stream=None):
        self.nch, self.nb, self.n = int(nch), int(nbasis), int(nch) * int(nbasis)
        lv = np.ascontiguousarray(lval, dtype=np.int32)
        et = np.ascontiguousarray(ethr, dtype=np.float64)
        assert lv.shape == (nch,) and et.shape == (nch,)
        self._h = C.c_void_p()
        self._stream = stream
        rc = lib().hprmat_setup(C.byref(self._h), C.c_int(nch), C.c_int(nbasis), C.c_double(a), C.c_double(h2m),
                                lv.ctypes.data_as(C.c_void_p), et.ctypes.data_as(C.c_void_p), C.c_int(max_mode),
                                _stream(stream))
        _check(rc, "hprmat_setup")

    @classmethod
    def sector(cls, nch, nbasis, a_lo, a_hi, h2m, lval, ethr, max_mode=0, stream=None):
        """hprmat_setup_sector: context of the sub-interval (a_lo, a_hi) of a propagation."""
        self = cls.__new__(cls)
        self.nch, self.nb, self.n = int(nch), int(nbasis), int(nch) * int(nbasis)
        lv = np.ascontiguousarray(lval, dtype=np.int32)
        et = np.ascontiguousarray(ethr, dtype=np.float64)
        self._h = C.c_void_p()
        self._stream = stream
        rc = lib().hprmat_setup_sector(C.byref(self._h), C.c_int(nch), C.c_int(nbasis), C.c_double(a_lo), C.c_double(a_hi),
                                       C.c_double(h2m), lv.ctypes.data_as(C.c_void_p), et.ctypes.data_as(C.c_void_p),
                                       C.c_int(max_mode), _stream(stream))
        _check(rc, "hprmat_setup_sector")
        return self

    def solve_sector(self, energy, V, mode=HPRMAT_FP64, max_refine=-1, tol=0.0, allow=(HPRMAT_OK,)):
        """hprmat_solve_sector: returns (Rsec, info); Rsec torch complex128 [4, nch, nch], block b holds the column-major
        matrix (use Rsec[b].T) in the order LL, LR, RL, RR."""
        assert V.is_cuda and V.dtype == torch.complex128 and V.is_contiguous() and V.numel() == self.nb * self.nch ** 2
        Rsec = torch.empty((4, self.nch, self.nch), dtype=torch.complex128, device=V.device)
        info = hprmat_info()
        rc = lib().hprmat_solve_sector(self._h, C.c_double(energy), _dev(V), C.c_int(mode), C.c_int(max_refine),
                                       C.c_double(tol), _dev(Rsec), C.byref(info))
        _check(rc, "hprmat_solve_sector", allow)
        return Rsec, info.as_dict()

    def mesh(self):
        r = np.zeros(self.nb)
        fa = np.zeros(self.nb)
        _check(lib().hprmat_mesh(self._h, r.ctypes.data_as(C.c_void_p), fa.ctypes.data_as(C.c_void_p)), "hprmat_mesh")
        return r, fa

    def solve(self, energy, V, mode=HPRMAT_FP64, max_refine=-1, tol=0.0, R=None, want_info=True, allow=(HPRMAT_OK,)):
        """hprmat_solve: V torch complex128 CUDA [nb, nch, nch]; returns (R [nch, nch] column-major as a torch tensor
        holding R^T in row-major terms -- use .T for R[c1, c2]), info dict or None)."""
        assert V.is_cuda and V.dtype == torch.complex128 and V.is_contiguous() and V.numel() == self.nb * self.nch ** 2
        if R is None:
            R = torch.empty((self.nch, self.nch), dtype=torch.complex128, device=V.device)
        info = hprmat_info() if want_info else None
        rc = lib().hprmat_solve(self._h, C.c_double(energy), _dev(V), C.c_int(mode), C.c_int(max_refine),
                                C.c_double(tol), _dev(R), C.byref(info) if want_info else None)
        _check(rc, "hprmat_solve", allow)
        return R, (info.as_dict() if want_info else None)

    def solve_nonlocal(self, energy, W, ldw=None, mode=HPRMAT_FP64, max_refine=-1, tol=0.0, R=None, want_info=True,
                       allow=(HPRMAT_OK,)):
        """hprmat_solve_nonlocal: W torch complex128 CUDA tensor whose memory is the column-major N x N matrix."""
        assert W.is_cuda and W.dtype == torch.complex128 and W.is_contiguous()
        ldw = self.n if ldw is None else int(ldw)
        assert W.numel() >= ldw * (self.n - 1) + self.n
        if R is None:
            R = torch.empty((self.nch, self.nch), dtype=torch.complex128, device=W.device)
        info = hprmat_info() if want_info else None
        rc = lib().hprmat_solve_nonlocal(self._h, C.c_double(energy), _dev(W), C.c_long(ldw), C.c_int(mode),
                                         C.c_int(max_refine), C.c_double(tol), _dev(R),
                                         C.byref(info) if want_info else None)
        _check(rc, "hprmat_solve_nonlocal", allow)
        return R, (info.as_dict() if want_info else None)

    def solve_host(self, energy, V_host, mode=HPRMAT_FP64, max_refine=-1, tol=0.0, R_host=None, allow=(HPRMAT_OK,)):
        """hprmat_solve_host: V and R are HOST buffers (numpy complex128); copies are inside the call."""
        V_host = np.ascontiguousarray(V_host, dtype=np.complex128)
        if R_host is None:
            R_host = np.empty((self.nch, self.nch), dtype=np.complex128)
        info = hprmat_info()
        rc = lib().hprmat_solve_host(self._h, C.c_double(energy), V_host.ctypes.data_as(C.c_void_p), C.c_int(mode),
                                     C.c_int(max_refine), C.c_double(tol), R_host.ctypes.data_as(C.c_void_p),
                                     C.byref(info))
        _check(rc, "hprmat_solve_host", allow)
        return R_host, info.as_dict()

    def set_option(self, option, value):
        """hprmat_set_option: per-context algorithm switches (0 = follow the process default)."""
        _check(lib().hprmat_set_option(self._h, C.c_int(option), C.c_int(value)), "hprmat_set_option")

    def last_status(self):
        """hprmat_last_status: (status code, refinement steps, pivot index) of the last solve; synchronises."""
        steps, piv = C.c_int(0), C.c_int(0)
        rc = lib().hprmat_last_status(self._h, C.byref(steps), C.byref(piv))
        if rc < 0:
            raise HprmatError(rc, "hprmat_last_status")
        return rc, steps.value, piv.value

    def graphs(self):
        """(captured, eager): launch sequences of this context replayed from CUDA graphs / left as plain launches."""
        a, b = C.c_int(0), C.c_int(0)
        _check(lib().hprmat_profile_graphs(self._h, C.byref(a), C.byref(b)), "hprmat_profile_graphs")
        return a.value, b.value

    def get_x(self, device="cuda"):
        X = torch.empty((self.nch, self.n), dtype=torch.complex128, device=device)  # column-major N x nch
        _check(lib().hprmat_get_x(self._h, _dev(X)), "hprmat_get_x")
        return X

    def get_matrix(self, energy, V):
        Cm = torch.empty((self.n, self.n), dtype=torch.complex128, device=V.device)  # column-major N x N
        _check(lib().hprmat_get_matrix(self._h, C.c_double(energy), _dev(V), _dev(Cm)), "hprmat_get_matrix")
        return Cm

    def destroy(self):
        if self._h:
            lib().hprmat_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


# ---- raw dense entries ----------------------------------------------------------------------------------------------
def hprmat_workspace_bytes(n, nrhs, mode=HPRMAT_FP64) -> int:
    return int(lib().hprmat_workspace_bytes(C.c_int(n), C.c_int(nrhs), C.c_int(mode)))


def _workspace(n, nrhs, mode, device):
    nbytes = hprmat_workspace_bytes(n, nrhs, mode)
    return torch.empty(nbytes + 256, dtype=torch.uint8, device=device), nbytes


def _aligned(ws):
    off = (-ws.data_ptr()) % 256
    return C.c_void_p(ws.data_ptr() + off)


def hprmat_zgemm(m, n, k, alpha, A, lda, B, ldb, beta, Cm, ldc, stream=None):
    rc = lib().hprmat_zgemm(_stream(stream), C.c_int(m), C.c_int(n), C.c_int(k), C.c_double(alpha), _dev(A),
                            C.c_int(lda), _dev(B), C.c_int(ldb), C.c_double(beta), _dev(Cm), C.c_int(ldc))
    _check(rc, "hprmat_zgemm")


def hprmat_fp64_algo(algo: int = 0) -> int:
    """Select (1: LU of C - E I, 2: LU of the block-preconditioned matrix) or query the FP64 factorisation of hprmat_solve."""
    return int(lib().hprmat_fp64_algo(C.c_int(algo)))


def hprmat_zgemm_algo(algo: int = 0) -> int:
    """Select (3 or 4) or query (anything else) the real decomposition of the complex128 GEMM."""
    return int(lib().hprmat_zgemm_algo(C.c_int(algo)))


def hprmat_cgemm_tf32(m, n, k, alpha, A_re, A_im, lda, B_re, B_im, ldb, beta, C_re, C_im, ldc, stream=None):
    """Planar complex64 GEMM on the tcgen05 TF32 tensor cores; all operands torch float32 CUDA tensors (column-major)."""
    rc = lib().hprmat_cgemm_tf32(_stream(stream), C.c_int(m), C.c_int(n), C.c_int(k), C.c_float(alpha), _dev(A_re),
                                 _dev(A_im), C.c_int(lda), _dev(B_re), _dev(B_im), C.c_int(ldb), C.c_float(beta),
                                 _dev(C_re), _dev(C_im), C.c_int(ldc))
    _check(rc, "hprmat_cgemm_tf32")


def hprmat_cgemm_3xtf32(m, n, k, alpha, A_re, A_im, lda, B_re, B_im, ldb, beta, C_re, C_im, ldc, stream=None):
    """Planar complex64 GEMM with FP32-class accuracy (3xTF32, mma.sync); operands as hprmat_cgemm_tf32."""
    rc = lib().hprmat_cgemm_3xtf32(_stream(stream), C.c_int(m), C.c_int(n), C.c_int(k), C.c_float(alpha), _dev(A_re),
                                   _dev(A_im), C.c_int(lda), _dev(B_re), _dev(B_im), C.c_int(ldb), C.c_float(beta),
                                   _dev(C_re), _dev(C_im), C.c_int(ldc))
    _check(rc, "hprmat_cgemm_3xtf32")


def hprmat_channel_functions(l, eta, x, is_open=True):
    """Host-only: (F, x dF/dx, G, x dG/dx) of an open channel or (0, 0, 1, x W'/W) of a closed one."""
    out = (C.c_double * 4)()
    rc = lib().hprmat_channel_functions(C.c_int(l), C.c_double(eta), C.c_double(x), C.c_int(1 if is_open else 0), out)
    _check(rc, "hprmat_channel_functions")
    return tuple(out)


def hprmat_collision_workspace_bytes(nch) -> int:
    return int(lib().hprmat_collision_workspace_bytes(C.c_int(nch)))


def hprmat_collision(lval, ethr, energy, h2m, a, R, zze2=None, info_dev=None, ws=None, stream=None):
    """Collision matrix of the open channels from the device R-matrix (zze2: per-channel Z1 Z2 e^2 in MeV fm, None =
    neutral).  R: torch complex128 CUDA tensor
    holding the column-major nch x nch matrix.  Returns (U, nopen): U a torch complex128 CUDA tensor of nopen*nopen
    elements (column-major) -- read U.view(nopen, nopen).T as the matrix."""
    nch = len(lval)
    if ws is None:
        ws = torch.empty(hprmat_collision_workspace_bytes(nch) + 256, dtype=torch.uint8, device=R.device)
    if info_dev is None:
        info_dev = torch.zeros(1, dtype=torch.int32, device=R.device)
    U = torch.empty(nch * nch, dtype=torch.complex128, device=R.device)
    lv = (C.c_int * nch)(*[int(v) for v in lval])
    et = (C.c_double * nch)(*[float(v) for v in ethr])
    nopen = C.c_int(0)
    zz = None if zze2 is None else (C.c_double * nch)(*[float(v) for v in zze2])
    rc = lib().hprmat_collision(_stream(stream), C.c_int(nch), lv, et, zz, C.c_double(energy), C.c_double(h2m), C.c_double(a),
                                _dev(R), _dev(U), C.byref(nopen), _dev(info_dev), _aligned(ws),
                                C.c_size_t(ws.numel() - 256))
    _check(rc, "hprmat_collision")
    return U[:nopen.value * nopen.value], nopen.value


def hprmat_propagate(a_lo, a_hi, R_in, Rsec, info_dev=None, ws=None, stream=None):
    """R-matrix at a_hi from the one at a_lo and the sector matrices (torch complex128 CUDA tensors, column-major)."""
    nch = R_in.shape[0]
    nbytes = int(lib().hprmat_propagate_workspace_bytes(C.c_int(nch)))
    if ws is None:
        ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=R_in.device)
    if info_dev is None:
        info_dev = torch.zeros(1, dtype=torch.int32, device=R_in.device)
    R_out = torch.empty((nch, nch), dtype=torch.complex128, device=R_in.device)
    rc = lib().hprmat_propagate(_stream(stream), C.c_int(nch), C.c_double(a_lo), C.c_double(a_hi), _dev(R_in), _dev(Rsec),
                                _dev(R_out), _dev(info_dev), _aligned(ws), C.c_size_t(ws.numel() - 256))
    _check(rc, "hprmat_propagate")
    return R_out


def hprmat_propagate_static_max_nch() -> int:
    return int(lib().hprmat_propagate_static_max_nch())


def hprmat_propagate_static(a_lo, a_hi, R_in, Rsec, R_out, info_dev, stream=None):
    """hprmat_propagate on the library's static device scratch (no allocation in the call; nch <= 128).  The caller passes
    every buffer, outputs included: R_out torch complex128 CUDA [nch, nch], info_dev torch int32 CUDA [1]."""
    nch = R_in.shape[0]
    rc = lib().hprmat_propagate_static(_stream(stream), C.c_int(nch), C.c_double(a_lo), C.c_double(a_hi), _dev(R_in),
                                       _dev(Rsec), _dev(R_out), _dev(info_dev))
    if rc == HPRMAT_ENOMEM:  # beyond the static limit: the library's message names it
        raise HprmatError(rc, "hprmat_propagate_static [" + lib().hprmat_last_cuda_error().decode() + "]")
    _check(rc, "hprmat_propagate_static")
    return R_out


def hprmat_zgetrf(n, A, lda, ipiv, info_dev, ws=None, stream=None):
    """In-place FP64 LU; A torch complex128 CUDA holding the column-major n x n matrix (lda >= n)."""
    if ws is None:
        ws, _ = _workspace(n, 0, HPRMAT_FP64, A.device)
    rc = lib().hprmat_zgetrf(_stream(stream), C.c_int(n), _dev(A), C.c_int(lda), _dev(ipiv), _dev(info_dev),
                             _aligned(ws), C.c_size_t(ws.numel() - 256))
    _check(rc, "hprmat_zgetrf")
    return ws


def hprmat_zgetrs(n, nrhs, A, lda, ipiv, B, ldb, ws, stream=None):
    rc = lib().hprmat_zgetrs(_stream(stream), C.c_int(n), C.c_int(nrhs), _dev(A), C.c_int(lda), _dev(ipiv), _dev(B),
                             C.c_int(ldb), _aligned(ws), C.c_size_t(ws.numel() - 256))
    _check(rc, "hprmat_zgetrs")


def hprmat_zsolve(n, nrhs, A, lda, B, ldb, ipiv=None, mode=HPRMAT_FP64, max_refine=-1, tol=0.0, ws=None, stream=None,
                  allow=(HPRMAT_OK,)):
    if ipiv is None:
        ipiv = torch.empty(max(n, 1), dtype=torch.int32, device=A.device)
    if ws is None:
        ws, _ = _workspace(n, nrhs, mode, A.device)
    info = hprmat_info()
    rc = lib().hprmat_zsolve(_stream(stream), C.c_int(n), C.c_int(nrhs), _dev(A), C.c_int(lda), _dev(B), C.c_int(ldb),
                             _dev(ipiv), C.c_int(mode), C.c_int(max_refine), C.c_double(tol), _aligned(ws),
                             C.c_size_t(ws.numel() - 256), C.byref(info))
    _check(rc, "hprmat_zsolve", allow)
    return ipiv, info.as_dict()
