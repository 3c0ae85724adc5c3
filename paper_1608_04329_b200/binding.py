"""ctypes binding of libhsp.so.  Names and arguments mirror include/hsp.h one to one; torch is
used only for device memory (`data_ptr()`) and the stream handle."""
import ctypes as C
import os
import re

import numpy as np

from . import build as _build

HSP_F32, HSP_F64 = 0, 1
HSP_OK, HSP_EINVAL, HSP_ENOMEM, HSP_ECUDA, HSP_ENOTPD, HSP_ENUMERIC = 0, -1, -2, -3, -4, -5
HSP_STORE_Z, HSP_FREEZE_SCALES, HSP_FREEZE_Z, HSP_FREEZE_BETA, HSP_NO_GRAPH, HSP_SERIAL = 1, 2, 4, 16, 32, 64
HSP_PAPER_DESIGN = 128

_HERE = os.path.dirname(os.path.abspath(__file__))
_HEADER = os.path.join(os.path.dirname(_HERE), "include", "hsp.h")
_lib = None


class HspError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"hsp error {code}: {msg}")
        self.code = code


def lib_path():
    return os.path.join(_HERE, "libhsp.so")


def declared_symbols():
    """Every function name include/hsp.h declares."""
    src = open(_HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(hsp_[a-z_0-9]+)\s*\(", src)))


def lib():
    """Load libhsp.so, building it with nvcc if it is missing or stale.  Fails loudly otherwise."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.build()
    L = C.CDLL(path)
    vp, ll, ull, dp = C.c_void_p, C.c_longlong, C.c_ulonglong, C.POINTER(C.c_double)
    L.hsp_create.argtypes = [C.POINTER(vp), vp, C.c_int, vp, ll, C.c_int, ull, vp]
    L.hsp_create_host.argtypes = [C.POINTER(vp), vp, C.c_int, vp, ll, C.c_int, ull, vp]
    L.hsp_sweep.argtypes = [vp, ll]
    L.hsp_reserve_history.argtypes = [vp, ll]
    L.hsp_create_shard.argtypes = [C.POINTER(vp), vp, C.c_int, vp, ll, C.c_int, ull, ll, vp]
    L.hsp_sweep_prepare.argtypes = [vp, ll]
    L.hsp_sweep_begin.argtypes = [vp]
    L.hsp_sweep_end.argtypes = [vp]
    L.hsp_xtz_device.argtypes = [vp]
    L.hsp_xtz_device.restype = vp
    L.hsp_gram_device.argtypes = [vp]
    L.hsp_gram_device.restype = vp
    L.hsp_get_draws.argtypes = [vp, vp, vp, vp]
    L.hsp_sync.argtypes = [vp]
    L.hsp_destroy.argtypes = [vp]
    L.hsp_last_error.restype = C.c_char_p
    L.hsp_get_latent.argtypes = [vp, vp, vp]
    L.hsp_get_state.argtypes = [vp, vp, vp, vp, vp, vp, C.POINTER(ll)]
    L.hsp_set_state.argtypes = [vp, vp, vp, vp, vp, vp, ll]
    L.hsp_set_flags.argtypes = [vp, C.c_uint]
    L.hsp_get_xtz.argtypes = [vp, vp]
    L.hsp_get_gram.argtypes = [vp, vp]
    L.hsp_get_chol.argtypes = [vp, vp]
    L.hsp_get_fused_pass_ms.argtypes = [vp, dp, C.POINTER(ll)]
    L.hsp_get_launch_count.argtypes = [vp]
    L.hsp_get_launch_count.restype = ll
    L.hsp_fused_variant.argtypes = [vp]
    L.hsp_fused_variant.restype = C.c_char_p
    L.hsp_dbg_philox.argtypes = [vp, vp, vp, ll, vp]
    L.hsp_dbg_uniform.argtypes = [ull, vp, C.c_uint, C.c_uint, vp, vp, ll, vp]
    L.hsp_dbg_tnpos.argtypes = [vp, vp, vp, ll, vp]
    L.hsp_dbg_norm_inv.argtypes = [vp, vp, ll, vp]
    L.hsp_dbg_cheng.argtypes = [C.c_double, ull, C.c_uint, vp, ll, vp]
    L.hsp_dbg_chol_trace.argtypes = [vp, vp, ll]
    L.hsp_get_plan.argtypes = [vp, C.POINTER(C.c_int), C.POINTER(C.c_int), C.POINTER(C.c_int), dp]
    L.hsp_set_option.argtypes = [vp, C.c_char_p, ll]
    L.hsp_get_option.argtypes = [vp, C.c_char_p, C.POINTER(ll)]
    L.hsp_set_output.argtypes = [vp, vp, vp, vp, ll]
    L.hsp_output_ready.argtypes = [vp, C.POINTER(ll)]
    L.hsp_output_wait.argtypes = [vp, C.POINTER(ll)]
    L.hsp_dbg_chol_trace.restype = ll
    L.hsp_xtz_noalloc.argtypes = [vp, C.c_int, vp, ll, C.c_int, ull, ll, vp, vp, vp, vp]
    L.hsp_noalloc_scratch_bytes.restype = ll
    L.hsp_noalloc_last_error.restype = C.c_char_p
    L.hsp_dbg_chol_schedule.argtypes = [C.c_int, C.c_int, C.c_int, vp, ll, dp]
    L.hsp_dbg_chol_schedule.restype = ll
    _lib = L
    return L


def _check(rc):
    if rc != HSP_OK:
        raise HspError(rc, lib().hsp_last_error().decode())


def _np(a):
    return a.ctypes.data_as(C.c_void_p)


def set_option(key, value):
    """hsp_set_option(NULL, key, value): process-wide default for chains created afterwards (value < 0: automatic)."""
    _check(lib().hsp_set_option(None, key.encode(), int(value)))


def reset_options():
    _check(lib().hsp_set_option(None, None, 0))


def get_option(key):
    v = C.c_longlong()
    _check(lib().hsp_get_option(None, key.encode(), C.byref(v)))
    return v.value


def _stream_handle(stream):
    import torch
    if stream is None:
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream), stream


class HorseshoeProbit:
    """hsp_create / hsp_sweep / hsp_get_draws on torch CUDA tensors (or host arrays with host=True)."""

    def __init__(self, X, y, seed, stream=None, host=False, row_offset=None):
        import torch
        L = lib()
        self._h = C.c_void_p()
        self.N, self.p = int(X.shape[0]), int(X.shape[1])
        self.n_last = 0
        sh, self._stream = _stream_handle(stream)
        if host:
            Xh = X if isinstance(X, torch.Tensor) else torch.from_numpy(np.ascontiguousarray(X))
            yh = y if isinstance(y, torch.Tensor) else torch.from_numpy(np.ascontiguousarray(y, dtype=np.uint8))
            assert not Xh.is_cuda and Xh.is_contiguous() and yh.dtype == torch.uint8
            dt = {torch.float32: HSP_F32, torch.float64: HSP_F64}[Xh.dtype]
            self._keep = (Xh, yh)
            _check(L.hsp_create_host(C.byref(self._h), Xh.data_ptr(), dt, yh.data_ptr(), self.N, self.p, seed, sh))
        else:
            assert X.is_cuda and y.is_cuda and X.is_contiguous() and y.is_contiguous() and y.dtype == torch.uint8
            dt = {torch.float32: HSP_F32, torch.float64: HSP_F64}[X.dtype]
            self._keep = (X, y)                       # borrowed by the library: keep alive
            if row_offset is None:
                _check(L.hsp_create(C.byref(self._h), X.data_ptr(), dt, y.data_ptr(), self.N, self.p, seed, sh))
            else:
                _check(L.hsp_create_shard(C.byref(self._h), X.data_ptr(), dt, y.data_ptr(), self.N, self.p, seed,
                                          int(row_offset), sh))

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            lib().hsp_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_flags(self, flags):
        _check(lib().hsp_set_flags(self._h, flags))

    def sweep(self, n_iter):
        _check(lib().hsp_sweep(self._h, n_iter))
        self.n_last = n_iter

    def reserve_history(self, n_iter):
        _check(lib().hsp_reserve_history(self._h, n_iter))

    def sync(self):
        _check(lib().hsp_sync(self._h))

    def stream_handle(self):
        """The cudaStream_t (as int) this chain enqueues on."""
        return int(self._stream.cuda_stream)

    def set_option(self, key, value):
        _check(lib().hsp_set_option(self._h, key.encode(), int(value)))

    # ---- asynchronous download of the draws into a pinned host ring (hsp_set_output)
    def set_output(self, beta, lam, tau, capacity):
        """beta [capacity, p], lam [capacity, p], tau [capacity]: pinned host tensors / arrays (any may be None)."""
        self._out = (beta, lam, tau)                   # borrowed by the library: keep alive
        ptrs = [None if t is None else (t.data_ptr() if hasattr(t, "data_ptr") else _np(t)) for t in self._out]
        _check(lib().hsp_set_output(self._h, *ptrs, int(capacity)))

    def output_ready(self):
        n = C.c_longlong()
        _check(lib().hsp_output_ready(self._h, C.byref(n)))
        return n.value

    def output_wait(self):
        n = C.c_longlong()
        _check(lib().hsp_output_wait(self._h, C.byref(n)))
        return n.value

    # ---- row-sharded chains: hsp_sweep_prepare / _begin / _end and the two buffers the caller all-reduces
    def sweep_prepare(self, n_iter):
        _check(lib().hsp_sweep_prepare(self._h, n_iter))
        self.n_last = n_iter

    def sweep_begin(self):
        _check(lib().hsp_sweep_begin(self._h))

    def sweep_end(self):
        _check(lib().hsp_sweep_end(self._h))

    def _device_view(self, ptr, shape):
        import torch

        class _Mem:                                   # zero-copy view of library memory (CUDA array interface)
            __cuda_array_interface__ = {"shape": shape, "typestr": "<f8", "data": (int(ptr), False), "version": 3}
        return torch.as_tensor(_Mem(), device=self._keep[0].device)

    def xtz_tensor(self):
        return self._device_view(lib().hsp_xtz_device(self._h), (self.p,))

    def gram_tensor(self):
        return self._device_view(lib().hsp_gram_device(self._h), (self.p, self.p))

    def get_draws(self, out=None):
        """(beta[n,p], lambda[n,p], tau[n]) of the last sweep() call as numpy arrays, or into the
        given tensors/arrays (host or device)."""
        n, p = self.n_last, self.p
        if out is None:
            beta, lam, tau = np.empty((n, p)), np.empty((n, p)), np.empty(n)
            _check(lib().hsp_get_draws(self._h, _np(beta), _np(lam), _np(tau)))
            return beta, lam, tau
        ptrs = [None if t is None else (t.data_ptr() if hasattr(t, "data_ptr") else _np(t)) for t in out]
        _check(lib().hsp_get_draws(self._h, *ptrs))
        return out

    def get_latent(self):
        z, side = np.empty(self.N), np.empty(self.N, dtype=np.int8)
        _check(lib().hsp_get_latent(self._h, _np(z), _np(side)))
        return z, side

    def get_state(self):
        p = self.p
        beta, lam, nu = np.empty(p), np.empty(p), np.empty(p)
        t, x, k = np.empty(1), np.empty(1), C.c_longlong()
        _check(lib().hsp_get_state(self._h, _np(beta), _np(lam), _np(nu), _np(t), _np(x), C.byref(k)))
        return dict(beta=beta, lam_inv2=lam, nu_inv=nu, tau_inv2=float(t[0]), xi_inv=float(x[0]), sweep=k.value)

    def set_state(self, beta=None, lam_inv2=None, nu_inv=None, tau_inv2=None, xi_inv=None, sweep=-1):
        def arr(a):
            return None if a is None else np.ascontiguousarray(a, dtype=np.float64)
        keep = [arr(beta), arr(lam_inv2), arr(nu_inv),
                None if tau_inv2 is None else np.array([tau_inv2], dtype=np.float64),
                None if xi_inv is None else np.array([xi_inv], dtype=np.float64)]
        _check(lib().hsp_set_state(self._h, *[None if a is None else _np(a) for a in keep], sweep))

    def _mat(self, fn, shape):
        out = np.empty(shape)
        _check(fn(self._h, _np(out)))
        return out

    def get_xtz(self):
        return self._mat(lib().hsp_get_xtz, self.p)

    def get_gram(self):
        return self._mat(lib().hsp_get_gram, (self.p, self.p))

    def get_chol(self):
        return np.tril(self._mat(lib().hsp_get_chol, (self.p, self.p)))

    def fused_pass_ms(self):
        ms, n = C.c_double(), C.c_longlong()
        _check(lib().hsp_get_fused_pass_ms(self._h, C.byref(ms), C.byref(n)))
        return ms.value, n.value

    def launch_count(self):
        return lib().hsp_get_launch_count(self._h)

    def fused_variant(self):
        return lib().hsp_fused_variant(self._h).decode()

    def plan(self):
        a, b, c, d = C.c_int(), C.c_int(), C.c_int(), C.c_double()
        _check(lib().hsp_get_plan(self._h, C.byref(a), C.byref(b), C.byref(c), C.byref(d)))
        return {"fused_ctas": a.value, "chol_ctas": b.value, "overlap": bool(c.value), "chol_est_us": d.value}

    def chol_trace(self):
        """Static tile schedule of rows c, d1 (and timestamps, with option chol_trace = 1): int64 [n_tasks, 12]."""
        n = lib().hsp_dbg_chol_trace(self._h, None, 0)
        if n < 0:
            _check(int(n))
        rows = np.zeros((n, 12), dtype=np.int64)
        n2 = lib().hsp_dbg_chol_trace(self._h, _np(rows), n)
        if n2 < 0:
            _check(int(n2))
        return rows


def xtz_noalloc(X, y, seed, k, beta, g_out, z_out=None, stream=None):
    """hsp_xtz_noalloc: torch CUDA tensors in, results written into the caller's g_out [p] (and z_out [N]) -- nothing is allocated."""
    import torch
    N, p = X.shape
    assert X.is_contiguous() and y.dtype == torch.uint8 and beta.dtype == torch.float64 and g_out.dtype == torch.float64
    dt = HSP_F32 if X.dtype == torch.float32 else HSP_F64
    rc = lib().hsp_xtz_noalloc(X.data_ptr(), dt, y.data_ptr(), N, p, int(seed), int(k), beta.data_ptr(), g_out.data_ptr(),
                               None if z_out is None else z_out.data_ptr(), _stream_handle(stream)[0])
    if rc != HSP_OK:
        raise HspError(rc, lib().hsp_noalloc_last_error().decode())


def noalloc_scratch_bytes():
    return int(lib().hsp_noalloc_scratch_bytes())


def chol_schedule(nt, sb, K):
    """Host-only: the static tile schedule of rows c, d1 for nt tile rows, inverse super-blocks of sb tiles, K CTAs:
    (int32 [n_tasks, 8] = {cta, type, i, j, kbeg, kend, slot_in, slot_out}, cost-model makespan in us)."""
    ms = C.c_double()
    n = lib().hsp_dbg_chol_schedule(nt, sb, K, None, 0, C.byref(ms))
    if n < 0:
        _check(int(n))
    rows = np.zeros((n, 8), dtype=np.int32)
    n2 = lib().hsp_dbg_chol_schedule(nt, sb, K, _np(rows), n, C.byref(ms))
    if n2 < 0:
        _check(int(n2))
    return rows, ms.value


# ---- device unit-test hooks (torch CUDA tensors in, torch CUDA tensors out) -------------------------
def dbg_philox(ctr, key):
    import torch
    n = ctr.shape[0]
    out = torch.empty((n, 4), dtype=torch.int32, device=ctr.device)
    _check(lib().hsp_dbg_philox(ctr.data_ptr(), key.data_ptr(), out.data_ptr(), n, _stream_handle(None)[0]))
    return out


def dbg_uniform(seed, idx, sweep, tag):
    import torch
    n = idx.shape[0]
    ua = torch.empty(n, dtype=torch.float64, device=idx.device)
    ub = torch.empty(n, dtype=torch.float64, device=idx.device)
    _check(lib().hsp_dbg_uniform(seed, idx.data_ptr(), sweep, tag, ua.data_ptr(), ub.data_ptr(), n, _stream_handle(None)[0]))
    return ua, ub


def dbg_tnpos(m, u):
    import torch
    w = torch.empty_like(m)
    _check(lib().hsp_dbg_tnpos(m.data_ptr(), u.data_ptr(), w.data_ptr(), m.numel(), _stream_handle(None)[0]))
    return w


def dbg_norm_inv(u):
    import torch
    x = torch.empty_like(u)
    _check(lib().hsp_dbg_norm_inv(u.data_ptr(), x.data_ptr(), u.numel(), _stream_handle(None)[0]))
    return x


def dbg_cheng(alpha, seed, sweep0, n, device="cuda"):
    import torch
    x = torch.empty(n, dtype=torch.float64, device=device)
    _check(lib().hsp_dbg_cheng(alpha, seed, sweep0, x.data_ptr(), n, _stream_handle(None)[0]))
    return x
