"""ctypes binding of oracle/libhsp_oracle.so (see hsp_oracle.cpp for what each call computes)."""
import ctypes as C

import numpy as np

from . import build as _build

F32, F64 = 0, 1
STORE_Z, FREEZE_SCALES, FREEZE_Z, LITERAL_Z, FREEZE_BETA, ROW_CHUNKS = 1, 2, 4, 8, 16, 32
TAG_Z, TAG_LAMBDA, TAG_TAU, TAG_E, TAG_NU, TAG_XI = 0, 1, 2, 3, 4, 5

_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        dp, u32p = C.POINTER(C.c_double), C.POINTER(C.c_uint32)
        L.hspo_philox4x32_10.argtypes = [u32p, u32p, u32p]
        L.hspo_philox4x32_10.restype = None
        L.hspo_uniforms.argtypes = [C.c_uint64, C.c_uint64, C.c_uint32, C.c_uint32, dp, dp]
        L.hspo_uniforms.restype = None
        for name in ("hspo_qinv", "hspo_norm_inv"):
            getattr(L, name).argtypes = [C.c_double]
            getattr(L, name).restype = C.c_double
        L.hspo_philox_many.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_longlong]
        L.hspo_philox_many.restype = None
        L.hspo_uniforms_many.argtypes = [C.c_uint64, C.c_void_p, C.c_uint32, C.c_uint32, C.c_void_p, C.c_void_p, C.c_longlong]
        L.hspo_uniforms_many.restype = None
        L.hspo_norm_inv_many.argtypes = [C.c_void_p, C.c_void_p, C.c_longlong]
        L.hspo_norm_inv_many.restype = None
        L.hspo_tnpos.argtypes = [C.c_double, C.c_double]
        L.hspo_tnpos.restype = C.c_double
        L.hspo_tnpos_many.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_longlong]
        L.hspo_tnpos_many.restype = None
        L.hspo_tnpos_rejection.argtypes = [C.c_double, C.c_uint64, C.c_uint64, C.c_uint32,
                                           C.POINTER(C.c_longlong)]
        L.hspo_tnpos_rejection.restype = C.c_double
        L.hspo_cheng_gamma.argtypes = [C.c_double, C.c_uint64, C.c_uint32, C.POINTER(C.c_longlong)]
        L.hspo_cheng_gamma.restype = C.c_double
        L.hspo_cholesky_lower.argtypes = [C.c_void_p, C.c_int]
        L.hspo_cholesky_lower.restype = C.c_int
        for name in ("hspo_solve_lower", "hspo_solve_lower_t"):
            getattr(L, name).argtypes = [C.c_void_p, C.c_int, C.c_void_p]
            getattr(L, name).restype = None
        L.hspo_create.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_longlong, C.c_int,
                                  C.c_ulonglong, C.c_void_p]
        L.hspo_create.restype = C.c_void_p
        L.hspo_destroy.argtypes = [C.c_void_p]
        L.hspo_destroy.restype = None
        L.hspo_set_flags.argtypes = [C.c_void_p, C.c_uint]
        L.hspo_sweep.argtypes = [C.c_void_p, C.c_longlong]
        L.hspo_get_draws.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.hspo_get_latent.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.hspo_set_latent.argtypes = [C.c_void_p, C.c_void_p]
        for name in ("hspo_get_xtz", "hspo_get_eta", "hspo_get_gram", "hspo_get_chol"):
            getattr(L, name).argtypes = [C.c_void_p, C.c_void_p]
        L.hspo_get_state.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, dp, dp,
                                     C.POINTER(C.c_longlong)]
        L.hspo_set_state.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, dp, dp,
                                     C.c_longlong]
        L.hspo_get_timing.argtypes = [C.c_void_p, dp, dp]
        L.hspo_get_literal_trials.argtypes = [C.c_void_p]
        L.hspo_get_literal_trials.restype = C.c_longlong
        L.hspo_max_threads.restype = C.c_int
        _lib = L
    return _lib


def max_threads():
    """Threads the timing-only ROW_CHUNKS mode uses."""
    return lib().hspo_max_threads()


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*[int(v) & 0xFFFFFFFF for v in ctr])
    k = (C.c_uint32 * 2)(*[int(v) & 0xFFFFFFFF for v in key])
    o = (C.c_uint32 * 4)()
    lib().hspo_philox4x32_10(c, k, o)
    return [int(v) for v in o]


def uniforms(seed, idx, sweep, tag):
    a, b = C.c_double(), C.c_double()
    lib().hspo_uniforms(seed, idx, sweep, tag, C.byref(a), C.byref(b))
    return a.value, b.value


def philox_many(ctr, key):
    ctr = np.ascontiguousarray(ctr, dtype=np.uint32)
    key = np.ascontiguousarray(key, dtype=np.uint32)
    out = np.empty_like(ctr)
    lib().hspo_philox_many(_ptr(ctr), _ptr(key), _ptr(out), ctr.shape[0])
    return out


def uniforms_many(seed, idx, sweep, tag):
    idx = np.ascontiguousarray(idx, dtype=np.uint64)
    ua, ub = np.empty(idx.size), np.empty(idx.size)
    lib().hspo_uniforms_many(seed, _ptr(idx), sweep, tag, _ptr(ua), _ptr(ub), idx.size)
    return ua, ub


def norm_inv_many(u):
    u = np.ascontiguousarray(u, dtype=np.float64)
    x = np.empty_like(u)
    lib().hspo_norm_inv_many(_ptr(u), _ptr(x), u.size)
    return x


def qinv(q):
    return lib().hspo_qinv(float(q))


def norm_inv(u):
    return lib().hspo_norm_inv(float(u))


def tnpos(m, u):
    return lib().hspo_tnpos(float(m), float(u))


def tnpos_many(m, u):
    m = np.ascontiguousarray(np.broadcast_to(np.asarray(m, dtype=np.float64), np.broadcast(m, u).shape))
    u = np.ascontiguousarray(np.broadcast_to(np.asarray(u, dtype=np.float64), m.shape))
    w = np.empty_like(m)
    lib().hspo_tnpos_many(_ptr(m), _ptr(u), _ptr(w), m.size)
    return w


def tnpos_rejection(m, seed, idx, sweep=1):
    n = C.c_longlong()
    w = lib().hspo_tnpos_rejection(float(m), seed, idx, sweep, C.byref(n))
    return w, n.value


def cheng_gamma(alpha, seed, sweep):
    t = C.c_longlong()
    x = lib().hspo_cheng_gamma(float(alpha), seed, sweep, C.byref(t))
    return x, t.value


def cholesky_lower(A):
    A = np.array(A, dtype=np.float64, order="C")
    rc = lib().hspo_cholesky_lower(_ptr(A), A.shape[0])
    return rc, np.tril(A)


def solve_lower(L, b, transpose=False):
    L = np.ascontiguousarray(L, dtype=np.float64)
    x = np.array(b, dtype=np.float64)
    (lib().hspo_solve_lower_t if transpose else lib().hspo_solve_lower)(_ptr(L), L.shape[0], _ptr(x))
    return x


class OracleChain:
    """The oracle's mirror of the C-ABI boundary (hsp_create / hsp_sweep / hsp_get_draws) on host arrays."""

    def __init__(self, X, y, seed, gram=None):
        X = np.ascontiguousarray(X)
        if X.dtype == np.float32:
            dt = F32
        elif X.dtype == np.float64:
            dt = F64
        else:
            raise TypeError("X must be float32 or float64")
        self.X = X
        self.y = np.ascontiguousarray(y, dtype=np.uint8)
        self.N, self.p = X.shape
        self.gram = None if gram is None else np.ascontiguousarray(gram, dtype=np.float64)
        self.h = lib().hspo_create(_ptr(self.X), dt, _ptr(self.y), self.N, self.p, seed, _ptr(self.gram))
        if not self.h:
            raise ValueError("hspo_create rejected its arguments")
        self.n_last = 0

    def close(self):
        if self.h:
            lib().hspo_destroy(self.h)
            self.h = None

    def __del__(self):
        self.close()

    def set_flags(self, flags):
        lib().hspo_set_flags(self.h, flags)

    def sweep(self, n_iter):
        rc = lib().hspo_sweep(self.h, n_iter)
        if rc != 0:
            raise RuntimeError(f"oracle sweep failed: {rc}")
        self.n_last = n_iter

    def get_draws(self):
        n, p = self.n_last, self.p
        beta, lam, tau = np.empty((n, p)), np.empty((n, p)), np.empty(n)
        lib().hspo_get_draws(self.h, _ptr(beta), _ptr(lam), _ptr(tau))
        return beta, lam, tau

    def get_latent(self):
        z, side = np.empty(self.N), np.empty(self.N, dtype=np.int8)
        lib().hspo_get_latent(self.h, _ptr(z), _ptr(side))
        return z, side

    def set_latent(self, z):
        z = np.ascontiguousarray(z, dtype=np.float64)
        assert z.shape == (self.N,)
        lib().hspo_set_latent(self.h, _ptr(z))

    def _vec(self, fn, shape):
        out = np.empty(shape)
        fn(self.h, _ptr(out))
        return out

    def get_xtz(self):
        return self._vec(lib().hspo_get_xtz, self.p)

    def get_eta(self):
        return self._vec(lib().hspo_get_eta, self.N)

    def get_gram(self):
        return self._vec(lib().hspo_get_gram, (self.p, self.p))

    def get_chol(self):
        return np.tril(self._vec(lib().hspo_get_chol, (self.p, self.p)))

    def get_state(self):
        p = self.p
        beta, lam, nu = np.empty(p), np.empty(p), np.empty(p)
        t, x, k = C.c_double(), C.c_double(), C.c_longlong()
        lib().hspo_get_state(self.h, _ptr(beta), _ptr(lam), _ptr(nu), C.byref(t), C.byref(x), C.byref(k))
        return dict(beta=beta, lam_inv2=lam, nu_inv=nu, tau_inv2=t.value, xi_inv=x.value, sweep=k.value)

    def set_state(self, beta=None, lam_inv2=None, nu_inv=None, tau_inv2=None, xi_inv=None, sweep=-1):
        def arr(a):
            return None if a is None else np.ascontiguousarray(a, dtype=np.float64)
        b, l, n = arr(beta), arr(lam_inv2), arr(nu_inv)
        t = None if tau_inv2 is None else C.byref(C.c_double(tau_inv2))
        x = None if xi_inv is None else C.byref(C.c_double(xi_inv))
        lib().hspo_set_state(self.h, _ptr(b), _ptr(l), _ptr(n), t, x, sweep)

    def get_timing(self):
        a, b = C.c_double(), C.c_double()
        lib().hspo_get_timing(self.h, C.byref(a), C.byref(b))
        return a.value, b.value

    def literal_trials(self):
        return lib().hspo_get_literal_trials(self.h)
