"""Thin ctypes binding of liblx.so (include/lx.h).  Same names as the C ABI; marshalling only.

PyTorch is used for device memory and streams, nothing else.  If the CUDA library is missing the import raises —
there is no fallback of any kind.
"""
import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.environ.get("LX_LIBRARY", os.path.join(_HERE, "liblx.so"))   # LX_LIBRARY: alternative build of liblx

if not os.path.exists(_SO):
    raise ImportError(f"{_SO} not found: build the CUDA library first (python -m paper_2210_03192_b200.build); "
                      "there is no CPU fallback")
_lib = C.CDLL(_SO)

LX_OK, LX_EINVAL, LX_EUNSUPPORTED, LX_ENOMEM, LX_ECUDA, LX_ENOTINIT, LX_ELIMIT, LX_ENOTPD = 0, -1, -2, -3, -4, -5, -6, -7
LX_MAX_L_AUX, LX_MAX_L_PRIM = 6, 4

EXPORTS = ["lx_init", "lx_finalize", "lx_strerror", "lx_version", "lx_eri3_batch", "lx_eri3_workspace_bytes",
           "lx_schedule_create", "lx_schedule_destroy", "lx_schedule_num_sets", "lx_schedule_num_integrals",
           "lx_df_workspace_bytes", "lx_df_gamma", "lx_df_J", "lx_eri3_batch_host", "lx_boys", "lx_launch_count", "lx_fp64_probe", "lx_kernel_family", "lx_kernel_family_k",
           "lx_cart_to_pure", "lx_solid_matrix", "lx_eri3_batch_pure", "lx_eri3_pure_workspace_bytes", "lx_async_status",
           "lx_schwarz_aux_host", "lx_schwarz_pair_host", "lx_eri3_batch_static", "lx_static_scratch_bytes",
           "lx_metric_2c", "lx_fit_solve"]


class lx_shells_t(C.Structure):
    _fields_ = [("nshell", C.c_int32), ("L", C.c_void_p), ("K", C.c_void_p), ("prim_off", C.c_void_p),
                ("center", C.c_void_p), ("zeta", C.c_void_p), ("coef", C.c_void_p), ("bf_off", C.c_void_p)]


_lib.lx_strerror.restype = C.c_char_p
_lib.lx_version.restype = C.c_char_p
_lib.lx_kernel_family.restype = C.c_char_p
_lib.lx_kernel_family.argtypes = [C.c_int] * 3
_lib.lx_kernel_family_k.restype = C.c_char_p
_lib.lx_kernel_family_k.argtypes = [C.c_int] * 4
_lib.lx_eri3_workspace_bytes.restype = C.c_size_t
_lib.lx_df_workspace_bytes.restype = C.c_size_t
_lib.lx_df_workspace_bytes.argtypes = [C.c_void_p]
_lib.lx_schedule_num_sets.restype = C.c_int64
_lib.lx_schedule_num_sets.argtypes = [C.c_void_p]
_lib.lx_schedule_num_integrals.restype = C.c_int64
_lib.lx_schedule_num_integrals.argtypes = [C.c_void_p]
_lib.lx_schedule_destroy.argtypes = [C.c_void_p]
_lib.lx_cart_to_pure.argtypes = [C.c_int, C.c_int64, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]
_lib.lx_solid_matrix.argtypes = [C.c_int, C.c_void_p]
_lib.lx_eri3_pure_workspace_bytes.restype = C.c_size_t
_lib.lx_eri3_pure_workspace_bytes.argtypes = [C.c_int] * 6
_lib.lx_eri3_batch_pure.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(lx_shells_t), C.POINTER(lx_shells_t), C.c_void_p,
                                    C.c_int, C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p]
_lib.lx_launch_count.restype = C.c_int64
_lib.lx_eri3_batch.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(lx_shells_t), C.POINTER(lx_shells_t),
                               C.c_void_p, C.c_int, C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p]
_lib.lx_eri3_batch_host.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(lx_shells_t), C.POINTER(lx_shells_t),
                                    C.c_void_p, C.c_int, C.c_void_p, C.c_int, C.c_void_p]
_lib.lx_eri3_workspace_bytes.argtypes = [C.c_int] * 6
_lib.lx_schedule_create.argtypes = [C.POINTER(lx_shells_t), C.POINTER(lx_shells_t), C.c_void_p, C.c_void_p,
                                    C.c_void_p, C.c_int, C.c_double, C.POINTER(C.c_void_p)]
_lib.lx_df_gamma.argtypes = [C.c_void_p, C.POINTER(lx_shells_t), C.POINTER(lx_shells_t), C.c_void_p, C.c_int,
                             C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p]
_lib.lx_df_J.argtypes = [C.c_void_p, C.POINTER(lx_shells_t), C.POINTER(lx_shells_t), C.c_void_p, C.c_void_p,
                         C.c_int, C.c_void_p, C.c_size_t, C.c_void_p]
_lib.lx_boys.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_void_p]


class LxError(RuntimeError):
    def __init__(self, status):
        self.status = status
        super().__init__(f"liblx status {status}: {_lib.lx_strerror(status).decode()}")


def _check(rc):
    if rc != LX_OK:
        raise LxError(rc)


def ncart(l):
    return (l + 1) * (l + 2) // 2


def lx_version():
    return _lib.lx_version().decode()


def lx_kernel_family(lx, la, lb):
    return _lib.lx_kernel_family(lx, la, lb).decode()


def lx_kernel_family_k(lx, la, lb, kmax):
    return _lib.lx_kernel_family_k(lx, la, lb, kmax).decode()


def lx_strerror(status):
    return _lib.lx_strerror(status).decode()


def lx_init(device=0):
    _check(_lib.lx_init(C.c_int(device)))


def lx_finalize():
    _check(_lib.lx_finalize())


def lx_async_status():
    """Status of the asynchronous work since the last call (LX_OK / LX_ENOMEM / LX_EINVAL); clears it."""
    return int(_lib.lx_async_status())


def lx_launch_count():
    return int(_lib.lx_launch_count())


def _stream_ptr(stream):
    if stream is None:
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream)


class HostShells:
    """lx_shells_t with HOST array members, from any object with the SoA attributes (e.g. lx_inputs.Shells)."""

    def __init__(self, t):
        self.L = np.ascontiguousarray(t.L, dtype=np.int32)
        self.K = np.ascontiguousarray(t.K, dtype=np.int32)
        self.prim_off = np.ascontiguousarray(t.prim_off, dtype=np.int32)
        self.center = np.ascontiguousarray(t.center, dtype=np.float64)
        self.zeta = np.ascontiguousarray(t.zeta, dtype=np.float64)
        self.coef = np.ascontiguousarray(t.coef, dtype=np.float64)
        self.bf_off = np.ascontiguousarray(t.bf_off, dtype=np.int32)
        self.nshell = len(self.L)
        self.struct = lx_shells_t(self.nshell, self.L.ctypes.data, self.K.ctypes.data, self.prim_off.ctypes.data,
                                  self.center.ctypes.data, self.zeta.ctypes.data, self.coef.ctypes.data,
                                  self.bf_off.ctypes.data)

    def nbytes(self):
        return sum(a.nbytes for a in (self.L, self.K, self.prim_off, self.center, self.zeta, self.coef))


class DeviceShells:
    """lx_shells_t with DEVICE array members (torch tensors own the memory)."""

    def __init__(self, t, device="cuda:0"):
        h = t if isinstance(t, HostShells) else HostShells(t)
        self.host = h
        self.device = torch.device(device)
        self.t = {k: torch.from_numpy(getattr(h, k)).to(self.device) for k in
                  ("L", "K", "prim_off", "center", "zeta", "coef", "bf_off")}
        self.nshell = h.nshell
        self.struct = lx_shells_t(self.nshell, *[self.t[k].data_ptr() for k in
                                                 ("L", "K", "prim_off", "center", "zeta", "coef", "bf_off")])


def _dev_i32(a, device):
    if isinstance(a, torch.Tensor):
        assert a.dtype == torch.int32 and a.is_cuda and a.is_contiguous()
        return a
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.int32)).to(device)


def lx_eri3_workspace_bytes(lx, la, lb, nx, npair, kmax_pair):
    return int(_lib.lx_eri3_workspace_bytes(lx, la, lb, nx, npair, kmax_pair))


def kmax_pair(prim_host, pair_idx):
    p = np.asarray(pair_idx).reshape(-1, 2)
    K = np.asarray(prim_host.K)
    return int(np.max(K[p[:, 0]] * K[p[:, 1]])) if len(p) else 1


def lx_eri3_batch(lx, la, lb, aux, prim, x_idx, pair_idx, out=None, workspace=None, stream=None, kmax=None):
    """(X|ab) for every listed pair × aux shell of one class → out[npair, nx, nc(lx), nc(la), nc(lb)] (device)."""
    dev = aux.device
    x_idx = _dev_i32(x_idx, dev)
    pair_idx = _dev_i32(pair_idx, dev).reshape(-1, 2)
    nx, npair = x_idx.numel(), pair_idx.shape[0]
    if kmax is None:
        kmax = kmax_pair(prim.host, pair_idx.cpu().numpy())
    if out is None:
        out = torch.empty((npair, nx, ncart(lx), ncart(la), ncart(lb)), dtype=torch.float64, device=dev)
    need = lx_eri3_workspace_bytes(lx, la, lb, nx, npair, kmax)
    if workspace is None:
        workspace = torch.empty(need, dtype=torch.uint8, device=dev)
    _check(_lib.lx_eri3_batch(lx, la, lb, C.byref(aux.struct), C.byref(prim.struct), x_idx.data_ptr(), nx,
                              pair_idx.data_ptr(), npair, out.data_ptr(), workspace.data_ptr(),
                              min(workspace.numel(), need), _stream_ptr(stream)))
    return out


_lib.lx_static_scratch_bytes.restype = C.c_size_t
_lib.lx_static_scratch_bytes.argtypes = []
_lib.lx_eri3_batch_static.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(lx_shells_t), C.POINTER(lx_shells_t), C.c_void_p, C.c_int,
                                      C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_void_p]


def lx_static_scratch_bytes():
    return int(_lib.lx_static_scratch_bytes())


def lx_eri3_batch_static(lx, la, lb, aux, prim, x_idx, pair_idx, out, kmax, stream=None):
    """lx_eri3_batch without a workspace and without any allocation in the library: the primitive-pair data lives in the
    library's static device array (4 MiB; LxError(LX_ELIMIT) beyond npair * kmax * 48 bytes).  `out`, `x_idx` and `pair_idx`
    must be device tensors the caller made (this wrapper allocates nothing either)."""
    assert isinstance(x_idx, torch.Tensor) and isinstance(pair_idx, torch.Tensor) and isinstance(out, torch.Tensor)
    assert x_idx.dtype == torch.int32 and pair_idx.dtype == torch.int32 and out.dtype == torch.float64
    assert x_idx.is_cuda and pair_idx.is_cuda and out.is_cuda and x_idx.is_contiguous() and pair_idx.is_contiguous() and out.is_contiguous()
    nx, npair = x_idx.numel(), pair_idx.numel() // 2
    assert out.numel() == npair * nx * ncart(lx) * ncart(la) * ncart(lb)
    _check(_lib.lx_eri3_batch_static(lx, la, lb, C.byref(aux.struct), C.byref(prim.struct), x_idx.data_ptr(), nx,
                                     pair_idx.data_ptr(), npair, int(kmax), out.data_ptr(), _stream_ptr(stream)))
    return out


def lx_eri3_batch_host(lx, la, lb, aux_host, prim_host, x_idx, pair_idx, out=None):
    """Host-buffer path: numpy in, numpy out; copies and synchronisation happen inside the library call."""
    x_idx = np.ascontiguousarray(x_idx, dtype=np.int32)
    pair_idx = np.ascontiguousarray(pair_idx, dtype=np.int32).reshape(-1, 2)
    nx, npair = len(x_idx), len(pair_idx)
    if out is None:
        out = np.empty((npair, nx, ncart(lx), ncart(la), ncart(lb)), dtype=np.float64)
    _check(_lib.lx_eri3_batch_host(lx, la, lb, C.byref(aux_host.struct), C.byref(prim_host.struct),
                                   x_idx.ctypes.data, nx, pair_idx.ctypes.data, npair, out.ctypes.data))
    return out


_lib.lx_schwarz_aux_host.argtypes = [C.POINTER(lx_shells_t), C.c_void_p]
_lib.lx_schwarz_pair_host.argtypes = [C.POINTER(lx_shells_t), C.c_void_p, C.c_int, C.c_void_p]


def lx_schwarz_aux_host(aux_host):
    """Q_X = sqrt(max_c (X_c|X_c)) per aux shell, evaluated on the GPU; HostShells in, numpy out."""
    q = np.zeros(aux_host.nshell, dtype=np.float64)
    _check(_lib.lx_schwarz_aux_host(C.byref(aux_host.struct), q.ctypes.data))
    return q


def lx_schwarz_pair_host(prim_host, pair_idx):
    """Q_ab = sqrt(max_ab (ab|ab)) per listed primary shell pair, evaluated on the GPU; HostShells in, numpy out."""
    pair_idx = np.ascontiguousarray(pair_idx, dtype=np.int32).reshape(-1, 2)
    q = np.zeros(len(pair_idx), dtype=np.float64)
    _check(_lib.lx_schwarz_pair_host(C.byref(prim_host.struct), pair_idx.ctypes.data, len(pair_idx), q.ctypes.data))
    return q


_lib.lx_metric_2c.argtypes = [C.POINTER(lx_shells_t), C.c_void_p, C.c_longlong]
_lib.lx_fit_solve.argtypes = [C.c_void_p, C.c_longlong, C.c_int, C.c_void_p, C.c_int, C.c_int]


def lx_metric_2c(aux_host, V=None):
    """Two-centre metric V[bf(X)+c, bf(Y)+c'] = (X_c|Y_c') of the aux basis on the current device; HostShells in,
    float64 CUDA tensor [naux_bf, naux_bf] out (written into `V` if given; its row stride is the leading dimension)."""
    n = int(sum((int(l) + 1) * (int(l) + 2) // 2 for l in aux_host.L))
    if V is None:
        V = torch.empty((n, n), dtype=torch.float64, device="cuda")
    assert V.is_cuda and V.dtype == torch.float64 and V.dim() == 2 and V.shape[0] >= n and V.stride(1) == 1
    _check(_lib.lx_metric_2c(C.byref(aux_host.struct), V.data_ptr(), V.stride(0)))
    return V


def lx_fit_solve(V, rhs, factored=False):
    """rhs <- V^-1 rhs in place (Cholesky; `V` [n, n] CUDA float64 is overwritten by its factor, `factored=True` reuses
    it).  rhs: CUDA float64 [n] or [nrhs, n] contiguous (one right-hand side per row), or None to factorise only."""
    n = V.shape[0]
    assert V.is_cuda and V.dtype == torch.float64 and V.dim() == 2 and V.shape[1] >= n and V.stride(1) == 1
    nrhs = 0
    if rhs is not None:
        assert rhs.is_cuda and rhs.dtype == torch.float64 and rhs.is_contiguous() and rhs.shape[-1] == n
        nrhs = rhs.numel() // n if n else 0
    _check(_lib.lx_fit_solve(V.data_ptr(), V.stride(0), n, rhs.data_ptr() if rhs is not None else None, nrhs,
                             1 if factored else 0))
    return rhs


class Schedule:
    """lx_schedule_t: class / contraction-degree buckets with Schwarz prefix lengths."""

    def __init__(self, aux_host, prim_host, q_aux, q_pair, pair_idx, tau):
        self.aux_host, self.prim_host = aux_host, prim_host
        pair_idx = np.ascontiguousarray(pair_idx, dtype=np.int32).reshape(-1, 2)
        qa = np.ascontiguousarray(q_aux, dtype=np.float64) if q_aux is not None else None
        qp = np.ascontiguousarray(q_pair, dtype=np.float64) if q_pair is not None else None
        h = C.c_void_p()
        _check(_lib.lx_schedule_create(C.byref(aux_host.struct), C.byref(prim_host.struct),
                                       qa.ctypes.data if qa is not None else None,
                                       qp.ctypes.data if qp is not None else None,
                                       pair_idx.ctypes.data, len(pair_idx), C.c_double(tau), C.byref(h)))
        self.handle = h

    @property
    def num_sets(self):
        return int(_lib.lx_schedule_num_sets(self.handle))

    @property
    def num_integrals(self):
        return int(_lib.lx_schedule_num_integrals(self.handle))

    @property
    def workspace_bytes(self):
        return int(_lib.lx_df_workspace_bytes(self.handle))

    def close(self):
        if self.handle is not None:
            _lib.lx_schedule_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def lx_df_gamma(sched, aux, prim, D, gamma=None, workspace=None, stream=None):
    """gamma_X = sum_ab (X|ab) D_ab over the unscreened sets of the schedule (device tensors)."""
    assert D.dtype == torch.float64 and D.is_cuda and D.stride(-1) == 1
    if gamma is None:
        gamma = torch.empty(int(aux.host.bf_off[-1]), dtype=torch.float64, device=D.device)
    if workspace is None:
        workspace = torch.empty(sched.workspace_bytes, dtype=torch.uint8, device=D.device)
    _check(_lib.lx_df_gamma(sched.handle, C.byref(aux.struct), C.byref(prim.struct), D.data_ptr(), D.stride(0),
                            gamma.data_ptr(), workspace.data_ptr(), workspace.numel(), _stream_ptr(stream)))
    return gamma


def lx_df_J(sched, aux, prim, d, J=None, workspace=None, stream=None):
    """J_ab = sum_X (X|ab) d_X over the unscreened sets of the schedule (device tensors)."""
    assert d.dtype == torch.float64 and d.is_cuda and d.is_contiguous()
    nbf = int(prim.host.bf_off[-1])
    if J is None:
        J = torch.empty((nbf, nbf), dtype=torch.float64, device=d.device)
    if workspace is None:
        workspace = torch.empty(sched.workspace_bytes, dtype=torch.uint8, device=d.device)
    _check(_lib.lx_df_J(sched.handle, C.byref(aux.struct), C.byref(prim.struct), d.data_ptr(), J.data_ptr(),
                        J.stride(0), workspace.data_ptr(), workspace.numel(), _stream_ptr(stream)))
    return J


def lx_eri3_batch_pure(lx, la, lb, aux, prim, x_idx, pair_idx, out=None, workspace=None, stream=None, kmax=None):
    """(X_m|ab) with solid-harmonic aux functions → out[npair, nx, 2lx+1, nc(la), nc(lb)] (device)."""
    dev = aux.device
    x_idx = _dev_i32(x_idx, dev)
    pair_idx = _dev_i32(pair_idx, dev).reshape(-1, 2)
    nx, npair = x_idx.numel(), pair_idx.shape[0]
    if kmax is None:
        kmax = kmax_pair(prim.host, pair_idx.cpu().numpy())
    if out is None:
        out = torch.empty((npair, nx, 2 * lx + 1, ncart(la), ncart(lb)), dtype=torch.float64, device=dev)
    need = int(_lib.lx_eri3_pure_workspace_bytes(lx, la, lb, nx, npair, kmax))
    if workspace is None:
        workspace = torch.empty(need, dtype=torch.uint8, device=dev)
    _check(_lib.lx_eri3_batch_pure(lx, la, lb, C.byref(aux.struct), C.byref(prim.struct), x_idx.data_ptr(), nx,
                                   pair_idx.data_ptr(), npair, kmax, out.data_ptr(), workspace.data_ptr(),
                                   C.c_size_t(workspace.numel()), _stream_ptr(stream)))
    return out


def lx_cart_to_pure(lx, cart, out=None, stream=None):
    """Cartesian → real solid-harmonic transform of the aux index: cart[npair, nx, nc(lx), na, nb] (device) →
    [npair, nx, 2lx+1, na, nb]."""
    assert cart.dtype == torch.float64 and cart.is_cuda and cart.is_contiguous() and cart.dim() == 5
    npair, nx, ncx, na, nb = cart.shape
    assert ncx == ncart(lx)
    if out is None:
        out = torch.empty((npair, nx, 2 * lx + 1, na, nb), dtype=torch.float64, device=cart.device)
    _check(_lib.lx_cart_to_pure(lx, C.c_int64(npair * nx), na * nb, cart.data_ptr(), out.data_ptr(), _stream_ptr(stream)))
    return out


def lx_solid_matrix(l):
    """The (2l+1) × nc(l) matrix lx_cart_to_pure applies (host; needs no device)."""
    m = np.zeros((2 * l + 1, ncart(l)), dtype=np.float64)
    _check(_lib.lx_solid_matrix(l, m.ctypes.data))
    return m


def lx_boys(T, mmax, stream=None):
    """F_m(T), m = 0..mmax, by the device routine the kernels use → [n, mmax+1]."""
    assert T.dtype == torch.float64 and T.is_cuda and T.is_contiguous()
    out = torch.empty((T.numel(), mmax + 1), dtype=torch.float64, device=T.device)
    _check(_lib.lx_boys(T.data_ptr(), T.numel(), mmax, out.data_ptr(), _stream_ptr(stream)))
    return out


def lx_fp64_probe(iters=20000):
    """Measured FP64 FMA rate of the device in TFLOP/s (register-resident DFMA chains)."""
    v = C.c_double(0.0)
    _check(_lib.lx_fp64_probe(C.c_int(iters), C.byref(v)))
    return float(v.value)
