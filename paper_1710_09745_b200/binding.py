"""Thin ctypes binding of libbkr.so (include/bkr.h).  Argument marshalling only: every step of the path
runs in the CUDA kernels behind the C ABI.  There is no CPU fallback: if the library is missing or no CUDA
device is present the calls raise.

Tensors are torch CUDA tensors used purely as device memory (``data_ptr()``); the stream is torch's current
stream at ``Context`` creation.  Function names mirror the C entry points (``bkr_dslash`` -> ``Context.dslash``).
"""
import ctypes
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libbkr.so")

F64, F32 = 0, 1
OK, EINVAL, ENOLINKS, ENOMEM, ECUDA, EBREAKDOWN, ENOCONV, ETOOBIG = 0, -1, -2, -3, -4, -5, -6, -7
MAX_N = 32
OPT_L2_BUDGET_MB, OPT_ROW_UNIT_TILES, OPT_ROW_VEC_POLICY, OPT_ABLATION = 0, 1, 2, 3
ABL_UNFUSED_UPDATES, ABL_UNFUSED_GRAM, ABL_VECTOR_BLAS, ABL_VECTOR_DSLASH = 1, 2, 4, 8
OPT_TUNE = 16  # + BKR_TUNE_* (bkr.h)
TUNE_F32_MATH = 4  # multi-BLAS on fp32 blocks: 0 FP64 tensor products (default), 1 split-TF32, 2 / 3 TF32 updates / reductions only
F32_MATH_FP64, F32_MATH_TF32, F32_MATH_TF32_UPDATES, F32_MATH_TF32_GRAM = 0, 1, 2, 3

SYMBOLS = (
    "bkr_create", "bkr_destroy", "bkr_load_links", "bkr_field_bytes", "bkr_pack", "bkr_unpack", "bkr_dslash", "bkr_dslash_xpay",
    "bkr_apply_M", "bkr_gram", "bkr_gram_static", "bkr_block_axpy", "bkr_block_update", "bkr_block_axpy_gram", "bkr_block_qpx_update", "bkr_cholesky_upper", "bkr_hpd_inverse", "bkr_solve_block",
    "bkr_solve_cg", "bkr_solve_block_host", "bkr_solve_cg_host", "bkr_bench_iterations", "bkr_last_cuda_error",
    "bkr_strerror", "bkr_version", "bkr_dslash_variant", "bkr_set_dslash_variant", "bkr_set_option", "bkr_microbench", "bkr_solver_state", "bkr_solve_many",
)


class Stats(ctypes.Structure):
    _fields_ = [("iters", ctypes.c_int), ("reliable_updates", ctypes.c_int), ("status", ctypes.c_int),
                ("restarts", ctypes.c_int), ("seconds", ctypes.c_double), ("true_relres_max", ctypes.c_double),
                ("iter_relres_max", ctypes.c_double), ("gpu_launches", ctypes.c_longlong),
                ("reorthonormalisations", ctypes.c_int)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


class BkrError(RuntimeError):
    def __init__(self, status, where, cuda=0):
        self.status = status
        msg = "%s: %s (%d)" % (where, lib().bkr_strerror(status).decode(), status)
        if cuda:
            msg += " [cudaError %d]" % cuda
        super().__init__(msg)


_lib = None


def lib():
    """Load libbkr.so.  Raises if it has not been built (python -m paper_1710_09745_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise FileNotFoundError("%s is missing: run `python -m paper_1710_09745_b200.build`" % LIB_PATH)
        L = ctypes.CDLL(LIB_PATH)
        vp, ci, cd = ctypes.c_void_p, ctypes.c_int, ctypes.c_double
        sig = {
            "bkr_create": (ci, [ctypes.POINTER(vp), ctypes.POINTER(ci), ci, vp]),
            "bkr_destroy": (ci, [vp]),
            "bkr_load_links": (ci, [vp, vp, vp, ci]),
            "bkr_field_bytes": (ctypes.c_size_t, [vp, ci, ci]),
            "bkr_pack": (ci, [vp, ci, ci, vp, vp]),
            "bkr_unpack": (ci, [vp, ci, ci, vp, vp]),
            "bkr_dslash": (ci, [vp, ci, ci, ci, vp, vp]),
            "bkr_dslash_xpay": (ci, [vp, ci, ci, ci, cd, vp, vp, vp]),
            "bkr_apply_M": (ci, [vp, cd, ci, ci, vp, vp]),
            "bkr_gram": (ci, [vp, ci, ci, vp, vp, ci, vp]),
            "bkr_gram_static": (ci, [vp, ci, ci, vp, vp, ci, vp]),
            "bkr_block_axpy": (ci, [vp, ci, ci, vp, vp, vp]),
            "bkr_block_update": (ci, [vp, ci, ci, ci, ci, vp, vp, vp, vp]),
            "bkr_block_axpy_gram": (ci, [vp, ci, ci, vp, vp, vp, vp]),
            "bkr_block_qpx_update": (ci, [vp, ci, ci, vp, vp, vp, vp, vp, vp, vp, ci, ci]),
            "bkr_cholesky_upper": (ci, [vp, ci, vp, vp, vp, vp]),
            "bkr_hpd_inverse": (ci, [vp, ci, vp, vp, vp]),
            "bkr_solve_block": (ci, [vp, cd, ci, vp, vp, cd, ci, ci, cd, vp, ctypes.POINTER(Stats)]),
            "bkr_solve_cg": (ci, [vp, cd, ci, vp, vp, cd, ci, ci, vp, vp, ctypes.POINTER(Stats)]),
            "bkr_solve_many": (ci, [vp, cd, ci, ci, vp, vp, cd, cd, ci, ci, cd, vp, ctypes.POINTER(Stats)]),
            "bkr_solve_block_host": (ci, [vp, cd, ci, vp, vp, cd, ci, ci, cd, vp, ctypes.POINTER(Stats)]),
            "bkr_solve_cg_host": (ci, [vp, cd, ci, vp, vp, cd, ci, ci, vp, vp, ctypes.POINTER(Stats)]),
            "bkr_bench_iterations": (ci, [vp, cd, ci, ci, vp, ci, ctypes.POINTER(ctypes.c_longlong)]),
            "bkr_last_cuda_error": (ci, [vp]),
            "bkr_strerror": (ctypes.c_char_p, [ci]),
            "bkr_version": (ctypes.c_char_p, []),
            "bkr_dslash_variant": (ci, [vp]),
            "bkr_set_dslash_variant": (ci, [vp, ci]),
            "bkr_set_option": (ci, [vp, ci, ci]),
            "bkr_solver_state": (ci, [vp, ctypes.POINTER(ci)]),
            "bkr_microbench": (ci, [vp, ci, ci, ctypes.POINTER(cd)]),
        }
        for name, (res, args) in sig.items():
            f = getattr(L, name)
            f.restype, f.argtypes = res, args
        _lib = L
    return _lib


def _dev_ptr(t, name):
    if not isinstance(t, torch.Tensor) or not t.is_cuda or not t.is_contiguous():
        raise TypeError("%s must be a contiguous CUDA tensor" % name)
    return ctypes.c_void_p(t.data_ptr())


class Context:
    """Owns a bkr_ctx for one lattice.  All tensor arguments are CUDA tensors on the context's device."""

    def __init__(self, dims, device=0):
        if not torch.cuda.is_available():
            raise RuntimeError("libbkr needs a CUDA device (sm_100a); there is no CPU fallback")
        self.dims = tuple(int(d) for d in dims)
        self.device = torch.device("cuda", int(device))
        self.V = 1
        for d in self.dims:
            self.V *= d
        self.Vh = self.V // 2
        self.L = 3 * self.Vh
        self._h = ctypes.c_void_p()
        stream = torch.cuda.current_stream(self.device).cuda_stream
        rc = lib().bkr_create(ctypes.byref(self._h), (ctypes.c_int * 4)(*self.dims), int(device),
                              ctypes.c_void_p(stream))
        if rc != OK:
            self._h = None
            raise BkrError(rc, "bkr_create")

    def close(self):
        if getattr(self, "_h", None) and _lib is not None:
            _lib.bkr_destroy(self._h)
        self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:  # interpreter shutdown: the library may already be gone
            pass

    def _check(self, rc, where, allow=()):
        if rc != OK and rc not in allow:
            raise BkrError(rc, where, lib().bkr_last_cuda_error(self._h))
        return rc

    # ---- links and layouts
    def load_links(self, fat, lng, also_f32=False):
        """fat, lng: (4, V, 3, 3) complex128 CUDA tensors (canonical layout)."""
        assert fat.dtype == torch.complex128 and lng.dtype == torch.complex128
        assert tuple(fat.shape) == (4, self.V, 3, 3) and tuple(lng.shape) == (4, self.V, 3, 3)
        self._check(lib().bkr_load_links(self._h, _dev_ptr(fat, "fat"), _dev_ptr(lng, "lng"), int(also_f32)),
                    "bkr_load_links")

    def field_bytes(self, N, prec=F64):
        return int(lib().bkr_field_bytes(self._h, int(N), int(prec)))

    def empty_native(self, N, prec=F64):
        """uninitialised native block [rhs][a][e] as a flat real tensor (fp64 or fp32)."""
        dt = torch.float64 if prec == F64 else torch.float32
        return torch.empty(self.L * int(N) * 2, dtype=dt, device=self.device)

    def pack(self, canonical, prec=F64, out=None):
        """(N, Vh, 3) complex128 -> native block."""
        N = self._n_of(canonical)
        out = self.empty_native(N, prec) if out is None else out
        self._check(lib().bkr_pack(self._h, N, int(prec), _dev_ptr(canonical, "canonical"), _dev_ptr(out, "native")),
                    "bkr_pack")
        return out

    def unpack(self, native, N, prec=F64, out=None):
        out = torch.empty((int(N), self.Vh, 3), dtype=torch.complex128, device=self.device) if out is None else out
        self._check(lib().bkr_unpack(self._h, int(N), int(prec), _dev_ptr(native, "native"), _dev_ptr(out, "canonical")),
                    "bkr_unpack")
        return out

    def _n_of(self, canonical):
        assert canonical.dtype == torch.complex128 and canonical.dim() == 3
        assert tuple(canonical.shape[1:]) == (self.Vh, 3), canonical.shape
        return int(canonical.shape[0])

    # ---- kernel-level calls on native blocks
    def dslash(self, out_parity, N, src, dst, prec=F64):
        self._check(lib().bkr_dslash(self._h, int(out_parity), int(N), int(prec), _dev_ptr(src, "in"), _dev_ptr(dst, "out")),
                    "bkr_dslash")
        return dst

    def dslash_xpay(self, out_parity, N, a, xp, src, dst, prec=F64):
        """dst = a * xp - D src (the second half of M, bkr.h)."""
        self._check(lib().bkr_dslash_xpay(self._h, int(out_parity), int(N), int(prec), float(a), _dev_ptr(xp, "xp"),
                                          _dev_ptr(src, "in"), _dev_ptr(dst, "out")), "bkr_dslash_xpay")
        return dst

    def apply_M(self, mass, N, src, dst, prec=F64):
        self._check(lib().bkr_apply_M(self._h, float(mass), int(N), int(prec), _dev_ptr(src, "in"), _dev_ptr(dst, "out")),
                    "bkr_apply_M")
        return dst

    def gram(self, N, X, Y, hermitian=False, prec=F64, out=None):
        K = torch.empty((int(N), int(N)), dtype=torch.complex128, device=self.device) if out is None else out
        self._check(lib().bkr_gram(self._h, int(N), int(prec), _dev_ptr(X, "X"), _dev_ptr(Y, "Y"), int(bool(hermitian)),
                                   _dev_ptr(K, "K")), "bkr_gram")
        return K

    def gram_static(self, N, X, Y, K, hermitian=False, prec=F64):
        """bkr_gram_static: K = X^dag Y into the caller's K without any allocation in the library (N <= 32, bkr.h)"""
        assert K.dtype == torch.complex128 and tuple(K.shape) == (int(N), int(N))
        self._check(lib().bkr_gram_static(self._h, int(N), int(prec), _dev_ptr(X, "X"), _dev_ptr(Y, "Y"), int(bool(hermitian)),
                                          _dev_ptr(K, "K")), "bkr_gram_static")
        return K

    def block_axpy(self, N, a, X, Y, prec=F64):
        assert a.dtype == torch.complex128 and tuple(a.shape) == (int(N), int(N))
        self._check(lib().bkr_block_axpy(self._h, int(N), int(prec), _dev_ptr(a, "a"), _dev_ptr(X, "X"), _dev_ptr(Y, "Y")),
                    "bkr_block_axpy")
        return Y

    def block_update(self, N, a, C, W, Z, precZ=F64, precW=F64, tri=0):
        """Z <- C + W a (C may be None); tri 0 general, 1 upper, 2 lower triangular a (bkr.h)."""
        assert a.dtype == torch.complex128 and tuple(a.shape) == (int(N), int(N))
        cptr = ctypes.c_void_p(0) if C is None else _dev_ptr(C, "C")
        self._check(lib().bkr_block_update(self._h, int(N), int(precZ), int(precW), int(tri), _dev_ptr(a, "a"), cptr,
                                           _dev_ptr(W, "W"), _dev_ptr(Z, "Z")), "bkr_block_update")
        return Z

    def block_axpy_gram(self, N, a, X, Y, prec=F64, out=None):
        """Y += X a and K = Y^dag Y of the updated Y in one pass; returns K (N x N complex128)."""
        assert a.dtype == torch.complex128 and tuple(a.shape) == (int(N), int(N))
        K = out if out is not None else torch.empty(int(N), int(N), dtype=torch.complex128, device=self.device)
        self._check(lib().bkr_block_axpy_gram(self._h, int(N), int(prec), _dev_ptr(a, "a"), _dev_ptr(X, "X"), _dev_ptr(Y, "Y"),
                                              _dev_ptr(K, "K")), "bkr_block_axpy_gram")
        return K

    def block_qpx_update(self, N, Sinv, Sdag, Wm, Q, P, Pn, X, prec=F64, do_qp=True, do_x=True):
        """Q <- Q Sinv, Pn <- Q + P Sdag (if do_qp) and X <- X + P Wm (if do_x) in one pass (bkr.h)."""
        for m in (Sinv, Sdag, Wm):
            assert m.dtype == torch.complex128 and tuple(m.shape) == (int(N), int(N))
        self._check(lib().bkr_block_qpx_update(self._h, int(N), int(prec), _dev_ptr(Sinv, "Sinv"), _dev_ptr(Sdag, "Sdag"),
                                               _dev_ptr(Wm, "Wm"), _dev_ptr(Q, "Q"), _dev_ptr(P, "P"), _dev_ptr(Pn, "Pn"),
                                               _dev_ptr(X, "X"), int(bool(do_qp)), int(bool(do_x))), "bkr_block_qpx_update")

    def cholesky_upper(self, H):
        N = int(H.shape[0])
        R, Ri = torch.empty_like(H), torch.empty_like(H)
        st = torch.zeros(1, dtype=torch.int32, device=self.device)
        self._check(lib().bkr_cholesky_upper(self._h, N, _dev_ptr(H, "H"), _dev_ptr(R, "R"), _dev_ptr(Ri, "Rinv"),
                                             _dev_ptr(st, "status")), "bkr_cholesky_upper")
        return R, Ri, int(st.item())

    def hpd_inverse(self, G):
        N = int(G.shape[0])
        Gi = torch.empty_like(G)
        st = torch.zeros(1, dtype=torch.int32, device=self.device)
        self._check(lib().bkr_hpd_inverse(self._h, N, _dev_ptr(G, "G"), _dev_ptr(Gi, "Ginv"), _dev_ptr(st, "status")),
                    "bkr_hpd_inverse")
        return Gi, int(st.item())

    # ---- canonical-layout conveniences built from the calls above (marshalling only)
    def dslash_canonical(self, out_parity, v, prec=F64):
        N = self._n_of(v)
        src = self.pack(v, prec)
        dst = self.empty_native(N, prec)
        self.dslash(out_parity, N, src, dst, prec)
        return self.unpack(dst, N, prec)

    def apply_M_canonical(self, mass, v, prec=F64):
        N = self._n_of(v)
        src = self.pack(v, prec)
        dst = self.empty_native(N, prec)
        self.apply_M(mass, N, src, dst, prec)
        return self.unpack(dst, N, prec)

    # ---- solvers (canonical fp64 device tensors)
    def solve_block(self, mass, B, X0=None, tol=1e-10, maxiter=10000, inner_prec=F64, delta=0.1, raise_on=()):
        N = self._n_of(B)
        X = torch.zeros_like(B) if X0 is None else X0.clone()
        rr = (ctypes.c_double * N)()
        st = Stats()
        rc = lib().bkr_solve_block(self._h, float(mass), N, _dev_ptr(B, "B"), _dev_ptr(X, "X"), float(tol), int(maxiter),
                                   int(inner_prec), float(delta), rr, ctypes.byref(st))
        self._check(rc, "bkr_solve_block", allow=(EBREAKDOWN, ENOCONV))
        return X, list(rr), st.as_dict()

    def solve_many(self, mass, B, N, tol_sloppy=5e-6, tol_fine=2e-9, X0=None, maxiter=10000, inner_prec=F64, delta=0.1):
        """nrhs = B.shape[0] right-hand sides in blocks of N, sloppy + fine sweep (bkr_solve_many).  Returns X, the true
        relative residuals after the last sweep and stats[block][sweep] as dicts."""
        nrhs = int(B.shape[0])
        X = torch.zeros_like(B) if X0 is None else X0.clone()
        rr = (ctypes.c_double * nrhs)()
        nb = nrhs // int(N)
        st = (Stats * (2 * nb))()
        rc = lib().bkr_solve_many(self._h, float(mass), nrhs, int(N), _dev_ptr(B, "B"), _dev_ptr(X, "X"), float(tol_sloppy),
                                  float(tol_fine), int(maxiter), int(inner_prec), float(delta), rr, st)
        self._check(rc, "bkr_solve_many", allow=(EBREAKDOWN, ENOCONV))
        return X, list(rr), [[st[2 * b + s].as_dict() for s in range(2)] for b in range(nb)]

    def solve_cg(self, mass, B, X0=None, tol=1e-10, maxiter=10000, batched=False):
        N = self._n_of(B)
        X = torch.zeros_like(B) if X0 is None else X0.clone()
        rr = (ctypes.c_double * N)()
        its = (ctypes.c_int * N)()
        st = Stats()
        rc = lib().bkr_solve_cg(self._h, float(mass), N, _dev_ptr(B, "B"), _dev_ptr(X, "X"), float(tol), int(maxiter),
                                int(bool(batched)), its, rr, ctypes.byref(st))
        self._check(rc, "bkr_solve_cg", allow=(ENOCONV,))
        return X, list(its), list(rr), st.as_dict()

    def solve_block_host(self, mass, B_host, X_host, tol=1e-10, maxiter=10000, inner_prec=F64, delta=0.1):
        """B_host, X_host: pinned (or pageable) CPU complex128 tensors (N, Vh, 3); X_host in/out."""
        N = self._n_of(B_host)
        assert not B_host.is_cuda and not X_host.is_cuda and B_host.is_contiguous() and X_host.is_contiguous()
        rr = (ctypes.c_double * N)()
        st = Stats()
        rc = lib().bkr_solve_block_host(self._h, float(mass), N, ctypes.c_void_p(B_host.data_ptr()),
                                        ctypes.c_void_p(X_host.data_ptr()), float(tol), int(maxiter), int(inner_prec),
                                        float(delta), rr, ctypes.byref(st))
        self._check(rc, "bkr_solve_block_host", allow=(EBREAKDOWN, ENOCONV))
        return list(rr), st.as_dict()

    def solve_cg_host(self, mass, B_host, X_host, tol=1e-10, maxiter=10000, batched=False):
        N = self._n_of(B_host)
        assert not B_host.is_cuda and not X_host.is_cuda and B_host.is_contiguous() and X_host.is_contiguous()
        rr = (ctypes.c_double * N)()
        its = (ctypes.c_int * N)()
        st = Stats()
        rc = lib().bkr_solve_cg_host(self._h, float(mass), N, ctypes.c_void_p(B_host.data_ptr()),
                                     ctypes.c_void_p(X_host.data_ptr()), float(tol), int(maxiter), int(bool(batched)),
                                     its, rr, ctypes.byref(st))
        self._check(rc, "bkr_solve_cg_host", allow=(ENOCONV,))
        return list(its), list(rr), st.as_dict()

    def bench_iterations(self, mass, B, iters, prec=F64):
        N = self._n_of(B)
        n = ctypes.c_longlong(0)
        self._check(lib().bkr_bench_iterations(self._h, float(mass), N, int(prec), _dev_ptr(B, "B"), int(iters),
                                               ctypes.byref(n)), "bkr_bench_iterations")
        return int(n.value)

    def solver_state(self):
        """dict(iters, done, breakdown, xpend) of the device-side loop flags (bkr.h)."""
        st = (ctypes.c_int * 4)()
        self._check(lib().bkr_solver_state(self._h, st), "bkr_solver_state")
        return {"iters": st[0], "done": st[1], "breakdown": st[2], "xpend": st[3]}

    def microbench(self, kind, reps=5):
        """(ms per launch, flop or bytes per launch) of the on-chip microbenchmark `kind` (bkr.h)."""
        r = (ctypes.c_double * 4)()
        self._check(lib().bkr_microbench(self._h, int(kind), int(reps), r), "bkr_microbench")
        return float(r[0]), float(r[1])

    def probe(self, kind):
        """on-chip probe `kind` (10..29, csrc/probes.cu): (SM cycles, work units per SM, second work count)"""
        r = (ctypes.c_double * 4)()
        self._check(lib().bkr_microbench(self._h, int(kind), 1, r), "bkr_microbench")
        return float(r[0]), float(r[1]), float(r[2])

    def set_option(self, option, value):
        """launch-policy knob (bkr.h BKR_OPT_*): OPT_L2_BUDGET_MB = 0, OPT_ROW_UNIT_TILES = 1; value 0 = default."""
        self._check(lib().bkr_set_option(self._h, int(option), int(value)), "bkr_set_option")

    def set_f32_math(self, mode):
        """tensor path of the multi-BLAS on fp32 blocks (bkr.h BKR_TUNE_F32_MATH): F32_MATH_FP64 (default) / _TF32 / _TF32_UPDATES / _TF32_GRAM"""
        self.set_option(OPT_TUNE + TUNE_F32_MATH, mode)

    def set_dslash_variant(self, variant):
        """-1 automatic, 0 plain, 1 window, 2 row-window stencil kernel for later calls (bkr.h)."""
        self._check(lib().bkr_set_dslash_variant(self._h, int(variant)), "bkr_set_dslash_variant")

    def dslash_variant(self):
        """0 = plain stencil kernel, 1 = shared-memory window kernel, 2 = row-window kernel, -1 = none yet (diagnostic)."""
        return int(lib().bkr_dslash_variant(self._h))


def version():
    return lib().bkr_version().decode()
