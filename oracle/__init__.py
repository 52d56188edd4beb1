"""ORACLE -- test infrastructure only (tests/, __graft_entry__.smoke(), bench.py's CPU legs).

ctypes binding of ``oracle/oracle.c``: a plain fp64 CPU statement of the hot path of
arXiv:1710.09745 (hop operator eq. 2, M = 4m^2 - D_eo D_oe, block BLAS eq. 3/4, thin QR
Alg. 2, CG, blockCGrQ Alg. 1, block reliable updates Alg. 3).  It never imports the CUDA
package and the CUDA package never imports it.  Arrays are numpy, complex128, C-contiguous:

    links   (4, V, 3, 3)    [mu][lexicographic site][row][col], phases/coefficients folded in
    vectors (N, Vh, 3)      [rhs][even-odd site index][colour]
    small   (N, N)          row-major
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")


def build(force=False):
    """Compile oracle.c with the host compiler (gcc -O2 -fopenmp).  No CUDA involved."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".%d.tmp" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None
_c = ctypes
_P = ctypes.c_void_p


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        for name in ("orc_dslash", "orc_dslash_sites", "orc_apply_M", "orc_cholesky_upper", "orc_hpd_inverse",
                     "orc_thin_qr", "orc_thin_qr2", "orc_cg", "orc_block_cg", "orc_block_cg_reorth", "orc_true_relres"):
            getattr(_lib, name).restype = ctypes.c_int
        _lib.orc_gram.restype = None
        _lib.orc_block_axpy.restype = None
        _lib.orc_upper_inverse.restype = None
    return _lib


def _ca(a):
    a = np.ascontiguousarray(a, dtype=np.complex128)
    return a


def _ptr(a):
    return a.ctypes.data_as(_P) if a is not None else None


def _dims(dims):
    return (ctypes.c_int * 4)(*[int(d) for d in dims])


def volume(dims):
    return int(np.prod([int(d) for d in dims]))


def dslash(dims, fat, lng, out_parity, v):
    """out = D_{out_parity, 1-out_parity} v   (eq. 2)."""
    fat, lng, v = _ca(fat), _ca(lng), _ca(v)
    out = np.empty_like(v)
    rc = lib().orc_dslash(_dims(dims), _ptr(fat), _ptr(lng), int(out_parity), int(v.shape[0]), _ptr(v), _ptr(out))
    if rc:
        raise ValueError("orc_dslash: %d" % rc)
    return out


def dslash_sites(dims, fat, lng, out_parity, v, e_idx):
    """D v at the listed output sites only -> (N, len(e_idx), 3)."""
    fat, lng, v = _ca(fat), _ca(lng), _ca(v)
    e = np.ascontiguousarray(e_idx, dtype=np.int64)
    out = np.empty((v.shape[0], e.size, 3), dtype=np.complex128)
    rc = lib().orc_dslash_sites(_dims(dims), _ptr(fat), _ptr(lng), int(out_parity), int(v.shape[0]), _ptr(v),
                                ctypes.c_long(e.size), e.ctypes.data_as(_P), _ptr(out))
    if rc:
        raise ValueError("orc_dslash_sites: %d" % rc)
    return out


def apply_M(dims, fat, lng, mass, v):
    """out = 4 m^2 v - D_eo D_oe v on even sites."""
    fat, lng, v = _ca(fat), _ca(lng), _ca(v)
    out, tmp = np.empty_like(v), np.empty_like(v)
    rc = lib().orc_apply_M(_dims(dims), _ptr(fat), _ptr(lng), ctypes.c_double(mass), int(v.shape[0]), _ptr(v),
                           _ptr(out), _ptr(tmp))
    if rc:
        raise ValueError("orc_apply_M: %d" % rc)
    return out


def _as_block(X):
    X = _ca(X)
    N = X.shape[0]
    L = X.size // N
    return X, N, L


def gram(X, Y):
    """K = X^dag Y (eq. 4); X, Y (N, ...) blocks; K (N, N)."""
    X, N, L = _as_block(X)
    Y, _, _ = _as_block(Y)
    K = np.empty((N, N), dtype=np.complex128)
    lib().orc_gram(ctypes.c_long(L), N, _ptr(X), _ptr(Y), _ptr(K))
    return K


def block_axpy(a, X, Y):
    """returns Y + X a (eq. 3); inputs are not modified."""
    X, N, L = _as_block(X)
    Y = _ca(Y).copy()
    a = _ca(a)
    lib().orc_block_axpy(ctypes.c_long(L), N, _ptr(a), _ptr(X), _ptr(Y))
    return Y


def cholesky_upper(H):
    H = _ca(H)
    N = H.shape[0]
    R = np.empty_like(H)
    rc = lib().orc_cholesky_upper(N, _ptr(H), _ptr(R))
    if rc:
        raise ArithmeticError("cholesky breakdown")
    return R


def upper_inverse(R):
    R = _ca(R)
    Ri = np.empty_like(R)
    lib().orc_upper_inverse(R.shape[0], _ptr(R), _ptr(Ri))
    return Ri


def hpd_inverse(G):
    G = _ca(G)
    Gi = np.empty_like(G)
    rc = lib().orc_hpd_inverse(G.shape[0], _ptr(G), _ptr(Gi))
    if rc:
        raise ArithmeticError("cholesky breakdown")
    return Gi


def thin_qr(Z, two_pass=False):
    """Algorithm 2: returns Q (same shape as Z), R (N, N) upper.  two_pass: orc_thin_qr2 (a second
    Cholesky-QR pass, shifted first pass on a failed pivot; refs [43, 44] of PAPER.md:184-186)."""
    Z, N, L = _as_block(Z)
    Q = Z.copy()
    R = np.empty((N, N), dtype=np.complex128)
    rc = (lib().orc_thin_qr2 if two_pass else lib().orc_thin_qr)(ctypes.c_long(L), N, _ptr(Q), _ptr(R))
    if rc:
        raise ArithmeticError("cholesky breakdown")
    return Q, R


def cg(dims, fat, lng, mass, b, x0=None, tol=1e-10, maxiter=10000):
    """textbook CG on M x = b for ONE rhs b (Vh, 3).  returns x, iters, status, hist."""
    fat, lng, b = _ca(fat), _ca(lng), _ca(b)
    x = np.zeros_like(b) if x0 is None else _ca(x0).copy()
    it = ctypes.c_int(0)
    hist = np.zeros(maxiter + 1)
    rc = lib().orc_cg(_dims(dims), _ptr(fat), _ptr(lng), ctypes.c_double(mass), _ptr(b), _ptr(x),
                      ctypes.c_double(tol), int(maxiter), ctypes.byref(it), hist.ctypes.data_as(_P))
    return x, it.value, rc, hist[: it.value + 1]


def block_cg(dims, fat, lng, mass, B, X0=None, tol=1e-10, maxiter=10000, mixed=False, delta=0.1, ntrace=0, reorth=False):
    """blockCGrQ (Algorithm 1; with mixed=True plus Algorithm 3).  B (N, Vh, 3).
    returns dict(X, iters, status, reliable_updates, hist, G, C, QP); G, C, QP = traces of the first ntrace iterations
    (P^dag M P, C after l.12, and Q^dag P right after l.8: PAPER.md:210).  reorth: every thin QR by two Cholesky-QR
    passes (orc_thin_qr2) -- for blocks with nearly dependent right-hand sides."""
    fat, lng, B = _ca(fat), _ca(lng), _ca(B)
    N = B.shape[0]
    X = np.zeros_like(B) if X0 is None else _ca(X0).copy()
    it, nup = ctypes.c_int(0), ctypes.c_int(0)
    hist = np.zeros(maxiter + 1)
    tG = np.zeros((max(ntrace, 1), N, N), dtype=np.complex128)
    tC = np.zeros((max(ntrace, 1), N, N), dtype=np.complex128)
    tQP = np.zeros((max(ntrace, 1), N, N), dtype=np.complex128)
    rc = (lib().orc_block_cg_reorth if reorth else lib().orc_block_cg)(_dims(dims), _ptr(fat), _ptr(lng), ctypes.c_double(mass), N, _ptr(B), _ptr(X),
                            ctypes.c_double(tol), int(maxiter), int(bool(mixed)), ctypes.c_double(delta),
                            ctypes.byref(it), ctypes.byref(nup), hist.ctypes.data_as(_P), int(ntrace), _ptr(tG),
                            _ptr(tC), _ptr(tQP))
    return dict(X=X, iters=it.value, status=rc, reliable_updates=nup.value, hist=hist[: it.value + 1],
                G=tG[:ntrace], C=tC[:ntrace], QP=tQP[:ntrace])


def true_relres(dims, fat, lng, mass, B, X):
    fat, lng, B, X = _ca(fat), _ca(lng), _ca(B), _ca(X)
    out = np.zeros(B.shape[0])
    rc = lib().orc_true_relres(_dims(dims), _ptr(fat), _ptr(lng), ctypes.c_double(mass), int(B.shape[0]), _ptr(B),
                               _ptr(X), out.ctypes.data_as(_P))
    if rc:
        raise ValueError("orc_true_relres: %d" % rc)
    return out
