"""Thin ctypes binding of the C-ABI library `libnd_b200.so` (include/nd_b200.h).

Argument marshalling only: every step of the hot path runs in the CUDA kernels behind the C calls.  PyTorch
supplies device memory (tensors) and the CUDA stream; numpy arrays are accepted for host-side canonical AoS fields.
There is no CPU fallback: if the library is missing it is built with nvcc, and if that fails or no CUDA device is
present the calls raise `NDError`.

Method names are the C names without the `nd_` prefix (Context.apply_Q <-> nd_apply_Q, ...).
"""
import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libnd_b200.so")

ND_OK = 0
ERROR_NAMES = {
    -1: "ND_ERR_BAD_ARG", -2: "ND_ERR_BAD_STATE", -3: "ND_ERR_NOT_SU3", -4: "ND_ERR_RECON8_SINGULAR",
    -5: "ND_ERR_CUDA", -6: "ND_ERR_NO_CONVERGENCE", -7: "ND_ERR_NOMEM",
}

_c_int, _c_dbl, _c_vp = ctypes.c_int, ctypes.c_double, ctypes.c_void_p
_c_ll, _c_ull, _c_sz = ctypes.c_longlong, ctypes.c_ulonglong, ctypes.c_size_t
_pd = ctypes.POINTER(ctypes.c_double)

# name -> (restype, argtypes): every symbol include/nd_b200.h declares
SIGNATURES = {
    "nd_create": (_c_int, [ctypes.POINTER(_c_vp), ctypes.POINTER(_c_int), _c_int, _c_int, _c_int, _c_int, _c_vp]),
    "nd_destroy": (_c_int, [_c_vp]),
    "nd_last_error": (ctypes.c_char_p, [_c_vp]),
    "nd_set_stream": (_c_int, [_c_vp, _c_vp]),
    "nd_volume": (_c_ll, [_c_vp]),
    "nd_spinor_bytes": (_c_sz, [_c_vp]),
    "nd_gauge_bytes": (_c_sz, [_c_vp]),
    "nd_launch_count": (_c_ll, [_c_vp]),
    "nd_shard_layout": (_c_int, [_c_int, _c_int, _c_int, ctypes.POINTER(_c_int), ctypes.POINTER(_c_int), ctypes.POINTER(_c_int),
                                 ctypes.POINTER(_c_int)]),
    "nd_set_sharding": (_c_int, [_c_vp, _c_int, _c_int, _c_vp, _c_vp, _c_vp, _c_vp]),
    "nd_set_halo_peers": (_c_int, [_c_vp, _c_vp, _c_vp, _c_vp]),
    "nd_halo_bytes": (_c_sz, [_c_vp]),
    "nd_halo_buffers": (_c_int, [_c_vp, ctypes.POINTER(_c_vp), ctypes.POINTER(_c_vp), ctypes.POINTER(_c_vp), ctypes.POINTER(_c_vp)]),
    "nd_set_stencil_variant": (_c_int, [_c_vp, _c_int]),
    "nd_get_stencil_variant": (_c_int, [_c_vp]),
    "nd_get_stencil_variant_for": (_c_int, [_c_vp, _c_int, _c_int]),
    "nd_set_gauge": (_c_int, [_c_vp, _c_vp, _c_int, _c_int]),
    "nd_get_gauge": (_c_int, [_c_vp, _c_vp, _c_int]),
    "nd_gauge_stats": (_c_int, [_c_vp, _pd]),
    "nd_pack_spinor": (_c_int, [_c_vp, _c_vp, _c_int, _c_int, _c_vp]),
    "nd_unpack_spinor": (_c_int, [_c_vp, _c_vp, _c_vp, _c_int, _c_int]),
    "nd_apply_Q": (_c_int, [_c_vp, _c_vp, _c_vp, _c_dbl]),
    "nd_apply_Q2": (_c_int, [_c_vp, _c_vp, _c_vp, _c_vp, _c_dbl]),
    "nd_apply_Q_axpbycz": (_c_int, [_c_vp, _c_vp, _c_vp, _c_dbl, _c_dbl, _c_dbl, _c_vp, _c_dbl, _c_vp, _c_dbl, _c_vp]),
    "nd_cheb_coeffs": (_c_int, [_c_int, _c_dbl, _pd, _pd]),
    "nd_minmax_coeffs": (_c_int, [_c_int, _c_dbl, _pd, _pd, _pd]),
    "nd_set_sign_poly": (_c_int, [_c_vp, _c_int, _pd, _c_dbl, _c_dbl, _c_dbl]),
    "nd_set_lowmodes": (_c_int, [_c_vp, _c_int, _c_vp, _pd]),
    "nd_apply_sign": (_c_int, [_c_vp, _c_vp, _c_vp, _c_vp, _c_int]),
    "nd_apply_DN": (_c_int, [_c_vp, _c_vp, _c_vp, _c_dbl, _c_vp, _c_int]),
    "nd_apply_sign_multi": (_c_int, [_c_vp, _c_int, _c_vp, _c_vp, _c_vp, _c_int]),
    "nd_apply_DN_multi": (_c_int, [_c_vp, _c_int, _c_vp, _c_vp, _c_dbl, _c_vp, _c_int]),
    "nd_apply_DNm": (_c_int, [_c_vp, _c_vp, _c_vp, _c_dbl, _c_dbl, _c_vp, _c_int]),
    "nd_solve_DNm": (_c_int, [_c_vp, _c_vp, _c_vp, _c_dbl, _c_dbl, _c_dbl, _c_int, _c_vp, _pd, ctypes.POINTER(_c_int)]),
    "nd_solve_DNm_mixed": (_c_int, [_c_vp, _c_vp, _c_vp, _c_vp, _c_dbl, _c_dbl, _c_dbl, _c_dbl, _c_int, _c_int, _c_vp, _c_vp, _pd,
                                    ctypes.POINTER(_c_int)]),
    "nd_convert_spinor": (_c_int, [_c_vp, _c_vp, _c_int, _c_vp, _c_int]),
    "nd_lowmodes_compute": (_c_int, [_c_vp, _c_int, _c_int, _c_int, _c_int, _c_dbl, _c_int, _c_dbl, _c_int, _c_ull, _c_vp, _pd, _pd,
                                     ctypes.POINTER(_c_int), _pd, _pd, _c_vp, ctypes.POINTER(_c_ll)]),
    "nd_lowmodes_work_spinors": (_c_sz, [_c_int, _c_int]),
    "nd_index_count": (_c_int, [_c_vp, _c_int, _c_int, _c_dbl, _c_int, _c_ull, ctypes.POINTER(_c_int), _pd, _pd, _c_vp,
                                ctypes.POINTER(_c_ll)]),
    "nd_index_work_spinors": (_c_sz, [_c_int]),
    "nd_choose_l": (_c_int, [_c_int, _pd, _c_int, _c_int, ctypes.POINTER(_c_int), _pd]),
    "nd_projector_error": (_c_int, [_c_int, _pd, _pd, _c_int, _pd, _pd, _pd, _pd]),
    "nd_heev": (_c_int, [_c_int, _pd, _pd, _pd]),
    "nd_axpy": (_c_int, [_c_vp, _pd, _c_vp, _c_vp]),
    "nd_scale": (_c_int, [_c_vp, _pd, _c_vp]),
    "nd_copy": (_c_int, [_c_vp, _c_vp, _c_vp]),
    "nd_dot": (_c_int, [_c_vp, _c_vp, _c_vp, _pd]),
    "nd_norm2": (_c_int, [_c_vp, _c_vp, _pd]),
    "nd_gamma5": (_c_int, [_c_vp, _c_vp, _c_vp]),
    "nd_block_dot": (_c_int, [_c_vp, _c_int, _c_vp, _c_vp, _pd]),
    "nd_block_axpy": (_c_int, [_c_vp, _c_int, _pd, _c_vp, _c_vp]),
    "nd_block_dot_dev": (_c_int, [_c_vp, _c_int, _c_vp, _c_vp, _c_vp]),
    "nd_block_axpy_dev": (_c_int, [_c_vp, _c_int, _c_vp, _c_vp, _c_vp]),
    "nd_dot_dev": (_c_int, [_c_vp, _c_vp, _c_vp, _c_vp]),
    "nd_norm2_dev": (_c_int, [_c_vp, _c_vp, _c_vp]),
    "nd_gaussian": (_c_int, [_c_vp, _c_vp, _c_ull]),
    "nd_dot_static": (_c_int, [_c_vp, _c_vp, _c_ll, _c_int, _c_int, _c_vp, _c_vp, ctypes.c_char_p, _c_sz]),
}

DOT_STATIC_MAX_SITES = 4194304          # ND_DOT_STATIC_MAX_SITES
DOT_STATIC_SCRATCH_BYTES = 262144       # ND_DOT_STATIC_SCRATCH_BYTES

EXCHANGE_START_FN = ctypes.CFUNCTYPE(_c_int, _c_vp, _c_vp, _c_vp, _c_vp, _c_vp, _c_sz)
EXCHANGE_WAIT_FN = ctypes.CFUNCTYPE(_c_int, _c_vp)
ALLREDUCE_FN = ctypes.CFUNCTYPE(_c_int, _c_vp, _c_vp, _c_int)

_lib = None


class NDError(RuntimeError):
    def __init__(self, code, message=""):
        self.code = code
        super().__init__(f"{ERROR_NAMES.get(code, code)}: {message}")


def load_library(build_if_missing=True):
    """dlopen libnd_b200.so (building it in-tree with nvcc first if it is absent) and set all prototypes."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        if not build_if_missing:
            raise NDError(-5, f"{LIB_PATH} not built")
        from . import build as _build

        _build.build()
    lib = ctypes.CDLL(LIB_PATH)
    for name, (res, args) in SIGNATURES.items():
        fn = getattr(lib, name)      # AttributeError if a declared symbol is missing: fail loudly
        fn.restype = res
        fn.argtypes = args
    _lib = lib
    return lib


def cheb_coeffs(n, eps):
    """nd_cheb_coeffs: (c[0..n], delta) - host utility, needs no GPU."""
    lib = load_library()
    c = np.zeros(n + 1, dtype=np.float64)
    delta = ctypes.c_double(0.0)
    rc = lib.nd_cheb_coeffs(int(n), float(eps), c.ctypes.data_as(_pd), ctypes.byref(delta))
    if rc != ND_OK:
        raise NDError(rc, "nd_cheb_coeffs")
    return c, delta.value


def minmax_coeffs(n, eps):
    """nd_minmax_coeffs: (c[0..n], delta, levelled error E) of the min-max polynomial of eq. 2.6 - host utility, no GPU."""
    lib = load_library()
    c = np.zeros(n + 1, dtype=np.float64)
    delta, lev = ctypes.c_double(0.0), ctypes.c_double(0.0)
    rc = lib.nd_minmax_coeffs(int(n), float(eps), c.ctypes.data_as(_pd), ctypes.byref(delta), ctypes.byref(lev))
    if rc != ND_OK:
        raise NDError(rc, "nd_minmax_coeffs")
    return c, delta.value, lev.value


def heev(a):
    """nd_heev: Hermitian eigendecomposition (cyclic Jacobi) of a k x k complex matrix -> (w ascending, Z columns) -
    host utility, needs no GPU."""
    lib = load_library()
    a = np.ascontiguousarray(a, dtype=np.complex128)
    k = a.shape[0]
    assert a.shape == (k, k)
    w = np.zeros(k)
    z = np.zeros((k, k), dtype=np.complex128)
    rc = lib.nd_heev(k, a.view(np.float64).ctypes.data_as(_pd), w.ctypes.data_as(_pd), z.view(np.float64).ctypes.data_as(_pd))
    if rc != ND_OK:
        raise NDError(rc, "nd_heev")
    return w, z


def projector_error(nu, rho, rest):
    """nd_projector_error: (kappa[2], bound[2], d[l]) of eq. 2.9-2.10 - host utility, needs no GPU."""
    lib = load_library()
    nu = np.ascontiguousarray(nu, dtype=np.float64)
    rho = np.ascontiguousarray(rho, dtype=np.float64)
    rest = np.ascontiguousarray(rest, dtype=np.float64)
    kappa, bound, d = np.zeros(2), np.zeros(2), np.zeros(len(nu))
    rc = lib.nd_projector_error(len(nu), nu.ctypes.data_as(_pd), rho.ctypes.data_as(_pd), len(rest),
                                rest.ctypes.data_as(_pd) if len(rest) else None, kappa.ctypes.data_as(_pd),
                                bound.ctypes.data_as(_pd), d.ctypes.data_as(_pd))
    if rc != ND_OK:
        raise NDError(rc, "nd_projector_error")
    return kappa, bound, d


def shard_layout(T, nranks, rank):
    """nd_shard_layout: (t_begin, t_local, crosses_seam_prev, crosses_seam_next) - host utility, needs no GPU."""
    lib = load_library()
    tb, tl, cp, cn = _c_int(0), _c_int(0), _c_int(0), _c_int(0)
    rc = lib.nd_shard_layout(int(T), int(nranks), int(rank), ctypes.byref(tb), ctypes.byref(tl), ctypes.byref(cp), ctypes.byref(cn))
    if rc != ND_OK:
        raise NDError(rc, "nd_shard_layout")
    return tb.value, tl.value, bool(cp.value), bool(cn.value)


def choose_l(abs_nu, l_min, l_max):
    """nd_choose_l: (l', gap) of the gap rule (R17) - host utility, needs no GPU."""
    lib = load_library()
    a = np.ascontiguousarray(abs_nu, dtype=np.float64)
    l, gap = ctypes.c_int(0), ctypes.c_double(0.0)
    rc = lib.nd_choose_l(len(a), a.ctypes.data_as(_pd), int(l_min), int(l_max), ctypes.byref(l), ctypes.byref(gap))
    if rc != ND_OK:
        raise NDError(rc, "nd_choose_l")
    return l.value, gap.value


def _ptr(x):
    """Device tensor / numpy array / int / None -> void*."""
    if x is None:
        return None
    if isinstance(x, np.ndarray):
        return x.ctypes.data
    if isinstance(x, int):
        return x
    return x.data_ptr()      # torch tensor


def dot_static(x, y, V, prec, out, device=0, stream=None):
    """nd_dot_static: out[0:2] = <x, y> (re, im) for two device SoA spinors of V sites, without a context and without
    any allocation - for callers that may not call cudaMalloc (memory owned by someone else's pool, allocator calls
    forbidden in the current phase, fixed memory budget).  The partial sums use a 256 KiB array inside the library image,
    shared by all calls on the device: keep calls that could overlap on one stream.  V <= DOT_STATIC_MAX_SITES.
    x, y, out: device tensors or raw device addresses; stream: a torch stream, a raw cudaStream_t or None."""
    lib = load_library()
    st = getattr(stream, "cuda_stream", stream)
    err = ctypes.create_string_buffer(512)
    rc = lib.nd_dot_static(_ptr(x), _ptr(y), int(V), int(prec), int(device), _c_vp(st), _ptr(out), err, len(err))
    if rc != ND_OK:
        raise NDError(rc, err.value.decode())


def _c2(a):
    a = complex(a)
    return (ctypes.c_double * 2)(a.real, a.imag)


class Context:
    """One lattice + gauge field on one GPU (nd_ctx).  Spinors are flat torch tensors of 24*V reals in the device
    SoA layout, made by `new_spinor` / `pack_spinor`."""

    def __init__(self, dims, prec=64, recon=12, bc_time=-1, device=0, stream=None):
        import torch

        self._torch = torch
        self.lib = load_library()
        self.dims = tuple(int(d) for d in dims)
        self.prec, self.recon, self.bc_time, self.device = int(prec), int(recon), int(bc_time), int(device)
        if not torch.cuda.is_available():
            raise NDError(-5, "no CUDA device: this library has no CPU fallback")
        self.torch_device = torch.device("cuda", self.device)
        torch.cuda.set_device(self.torch_device)
        # a dedicated non-default stream: CUDA-graph capture is impossible on the legacy default stream
        self.stream = stream if stream is not None else torch.cuda.Stream(device=self.torch_device)
        self.real_dtype = torch.float32 if self.prec == 32 else torch.float64
        self._h = _c_vp()
        cd = (_c_int * 4)(*self.dims)
        rc = self.lib.nd_create(ctypes.byref(self._h), cd, self.prec, self.recon, self.bc_time, self.device,
                                _c_vp(self.stream.cuda_stream))
        if rc != ND_OK:
            self._h = None
            raise NDError(rc, "nd_create failed (no CUDA device / bad arguments)")
        self.V = int(self.lib.nd_volume(self._h))
        self.spinor_bytes = int(self.lib.nd_spinor_bytes(self._h))
        self._keep = {}

    # -- plumbing
    def _chk(self, rc):
        if rc != ND_OK:
            raise NDError(rc, self.lib.nd_last_error(self._h).decode())

    def close(self):
        if getattr(self, "_h", None):
            self.lib.nd_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def synchronize(self):
        self.stream.synchronize()

    def new_spinor(self, count=None):
        """Uninitialised device spinor(s): flat [24 V] (or [count, 24 V]) tensor of the context's real type."""
        torch = self._torch
        shape = (24 * self.V,) if count is None else (int(count), 24 * self.V)
        with torch.cuda.stream(self.stream):
            return torch.empty(shape, dtype=self.real_dtype, device=self.torch_device)

    # -- domain decomposition
    def set_sharding(self, rank, nranks, start=None, wait=None, allreduce=None):
        """start(send_next, send_prev, recv_prev, recv_next, bytes), wait(), allreduce(d_buf, n): Python callables working on
        raw device pointers (ints); exceptions become a non-zero status.  nranks = 1 removes the sharding."""
        def guard(fn):
            def call(*a):
                try:
                    fn(*a[1:])          # drop the unused `user` pointer
                    return 0
                except Exception:       # a callback must not unwind into C
                    import traceback

                    traceback.print_exc()
                    return 1
            return call

        if nranks > 1:
            self._cb = (EXCHANGE_START_FN(guard(start)) if start is not None else None, EXCHANGE_WAIT_FN(guard(wait)),
                        ALLREDUCE_FN(guard(allreduce)))
            self._chk(self.lib.nd_set_sharding(self._h, int(rank), int(nranks),
                                               ctypes.cast(self._cb[0], _c_vp) if start is not None else None,
                                               ctypes.cast(self._cb[1], _c_vp), ctypes.cast(self._cb[2], _c_vp), None))
        else:
            self._chk(self.lib.nd_set_sharding(self._h, 0, 1, None, None, None, None))
            self._cb = None

    def set_halo_peers(self, recv_own, recv_of_next, recv_of_prev):
        """Peer-to-peer face exchange (nd_set_halo_peers): raw device pointers (ints) of the three receive windows of
        4 * halo_bytes() bytes each, or three None for the callback transfers."""
        self._chk(self.lib.nd_set_halo_peers(self._h, recv_own, recv_of_next, recv_of_prev))

    def halo_bytes(self):
        return int(self.lib.nd_halo_bytes(self._h))

    def halo_buffers(self):
        """(send_next, send_prev, recv_prev, recv_next) device pointers."""
        p = [_c_vp() for _ in range(4)]
        self._chk(self.lib.nd_halo_buffers(self._h, *[ctypes.byref(x) for x in p]))
        return tuple(int(x.value) for x in p)

    def wrap_device_memory(self, ptr, nbytes, dtype):
        """A torch tensor aliasing `nbytes` of device memory at `ptr` (owned by the library)."""
        torch = self._torch

        class _Raw:
            pass

        raw = _Raw()
        itemsize = torch.empty((), dtype=dtype).element_size()
        typestr = {torch.float32: "<f4", torch.float64: "<f8", torch.uint8: "|u1"}[dtype]
        raw.__cuda_array_interface__ = {"shape": (nbytes // itemsize,), "typestr": typestr, "data": (int(ptr), False), "version": 2}
        return torch.as_tensor(raw, device=self.torch_device)

    STENCIL = {"auto": 0, "site": 1, "tile": 2, "tile_tma": 3, "tile4": 4}

    def set_stencil_variant(self, name):
        self._chk(self.lib.nd_set_stencil_variant(self._h, self.STENCIL[name]))

    def get_stencil_variant(self):
        v = int(self.lib.nd_get_stencil_variant(self._h))
        return {n: k for k, n in self.STENCIL.items()}[v]

    def get_stencil_variant_for(self, fused_epilogue=False, nrhs=1):
        """The variant one call runs (plain / fused-epilogue stencil on nrhs right-hand sides): the dispatch's own choice."""
        v = int(self.lib.nd_get_stencil_variant_for(self._h, int(bool(fused_epilogue)), int(nrhs)))
        if v < 0:
            raise NDError(v, "nd_get_stencil_variant_for")
        return {n: k for k, n in self.STENCIL.items()}[v]

    def launch_count(self):
        return int(self.lib.nd_launch_count(self._h))

    def gauge_bytes(self):
        return int(self.lib.nd_gauge_bytes(self._h))

    # -- gauge
    def set_gauge(self, U):
        """U: numpy complex64/128 [4, L0, L1, L2, L3, 3, 3] (host) or a torch complex tensor on the device."""
        if isinstance(U, np.ndarray):
            U = np.ascontiguousarray(U)
            assert U.shape == (4,) + self.dims + (3, 3), U.shape
            prec = {np.dtype(np.complex64): 32, np.dtype(np.complex128): 64}[U.dtype]
            self._chk(self.lib.nd_set_gauge(self._h, U.ctypes.data, prec, 0))
        else:
            torch = self._torch
            U = U.contiguous()
            prec = {torch.complex64: 32, torch.complex128: 64}[U.dtype]
            self.stream.wait_stream(torch.cuda.current_stream(self.torch_device))
            self._chk(self.lib.nd_set_gauge(self._h, U.data_ptr(), prec, 1))

    def get_gauge(self):
        out = np.empty((4,) + self.dims + (3, 3), dtype=np.complex128)
        self._chk(self.lib.nd_get_gauge(self._h, out.ctypes.data, 0))
        return out

    def gauge_stats(self):
        out = (ctypes.c_double * 4)()
        self._chk(self.lib.nd_gauge_stats(self._h, out))
        return tuple(out)

    # -- layout
    def pack_spinor(self, psi, out=None):
        """psi: numpy complex [L0,L1,L2,L3,4,3] (host) -> device SoA tensor."""
        psi = np.ascontiguousarray(psi)
        assert psi.shape == self.dims + (4, 3), psi.shape
        prec = {np.dtype(np.complex64): 32, np.dtype(np.complex128): 64}[psi.dtype]
        if out is None:
            out = self.new_spinor()
        self._chk(self.lib.nd_pack_spinor(self._h, psi.ctypes.data, prec, 0, out.data_ptr()))
        self.synchronize()       # the pageable host source must stay alive until the copy is done
        return out

    def unpack_spinor(self, soa, prec=64):
        out = np.empty(self.dims + (4, 3), dtype=np.complex128 if prec == 64 else np.complex64)
        self._chk(self.lib.nd_unpack_spinor(self._h, soa.data_ptr(), out.ctypes.data, prec, 0))
        return out

    def pack_spinor_host(self, host_ptr, aos_prec, out):
        """Raw host pointer variant (pinned buffers in bench.py): asynchronous."""
        self._chk(self.lib.nd_pack_spinor(self._h, host_ptr, aos_prec, 0, out.data_ptr()))

    def unpack_spinor_host(self, soa, host_ptr, aos_prec):
        self._chk(self.lib.nd_unpack_spinor(self._h, soa.data_ptr(), host_ptr, aos_prec, 0))

    # -- operators
    def apply_Q(self, out, inp, m):
        self._chk(self.lib.nd_apply_Q(self._h, out.data_ptr(), inp.data_ptr(), float(m)))

    def apply_Q2(self, out, inp, tmp, m):
        self._chk(self.lib.nd_apply_Q2(self._h, out.data_ptr(), inp.data_ptr(), tmp.data_ptr(), float(m)))

    def apply_Q_axpbycz(self, out, inp, m, s0, s1=0.0, v1=None, s2=0.0, v2=None, s3=0.0, v3=None):
        self._chk(self.lib.nd_apply_Q_axpbycz(self._h, out.data_ptr(), inp.data_ptr(), float(m), float(s0),
                                              float(s1), _ptr(v1), float(s2), _ptr(v2), float(s3), _ptr(v3)))

    # -- sign / D_N
    def set_sign_poly(self, c, eps, qnorm, m):
        c = np.ascontiguousarray(c, dtype=np.float64)
        self._chk(self.lib.nd_set_sign_poly(self._h, len(c) - 1, c.ctypes.data_as(_pd), float(eps), float(qnorm), float(m)))

    def set_lowmodes(self, u, nu):
        """u: [l, 24 V] device tensor (kept alive by the context), nu: l Ritz values."""
        if u is None or len(nu) == 0:
            self._keep.pop("u", None)
            self._chk(self.lib.nd_set_lowmodes(self._h, 0, None, None))
            return
        nu = np.ascontiguousarray(nu, dtype=np.float64)
        assert u.is_contiguous() and u.shape == (len(nu), 24 * self.V)
        self._keep["u"] = u
        self._chk(self.lib.nd_set_lowmodes(self._h, len(nu), u.data_ptr(), nu.ctypes.data_as(_pd)))

    def apply_sign(self, out, inp, work, use_graph=False):
        assert work.is_contiguous() and work.numel() >= 3 * 24 * self.V
        self._chk(self.lib.nd_apply_sign(self._h, out.data_ptr(), inp.data_ptr(), work.data_ptr(), int(use_graph)))

    def apply_DN(self, out, inp, prefactor, work, use_graph=False):
        assert work.is_contiguous() and work.numel() >= 3 * 24 * self.V
        self._chk(self.lib.nd_apply_DN(self._h, out.data_ptr(), inp.data_ptr(), float(prefactor), work.data_ptr(),
                                       int(use_graph)))

    def apply_sign_multi(self, out, inp, work, use_graph=False):
        """out, inp: [nrhs, 24 V]; work: 3 * nrhs spinors."""
        nrhs = inp.shape[0]
        assert out.shape == inp.shape and out.is_contiguous() and inp.is_contiguous() and work.numel() >= 3 * nrhs * 24 * self.V
        self._chk(self.lib.nd_apply_sign_multi(self._h, nrhs, out.data_ptr(), inp.data_ptr(), work.data_ptr(), int(use_graph)))

    def apply_DN_multi(self, out, inp, prefactor, work, use_graph=False):
        nrhs = inp.shape[0]
        assert out.shape == inp.shape and out.is_contiguous() and inp.is_contiguous() and work.numel() >= 3 * nrhs * 24 * self.V
        self._chk(self.lib.nd_apply_DN_multi(self._h, nrhs, out.data_ptr(), inp.data_ptr(), float(prefactor), work.data_ptr(),
                                             int(use_graph)))

    def apply_DNm(self, out, inp, prefactor, mq, work, use_graph=False):
        assert work.is_contiguous() and work.numel() >= 3 * 24 * self.V
        self._chk(self.lib.nd_apply_DNm(self._h, out.data_ptr(), inp.data_ptr(), float(prefactor), float(mq),
                                        work.data_ptr(), int(use_graph)))

    def solve_DNm(self, x, b, prefactor, mq, tol=1e-8, maxit=500, work=None):
        """-> (relres, iters, converged); x is overwritten with the solution."""
        if work is None:
            work = self.new_spinor(8)
        assert work.is_contiguous() and work.numel() >= 8 * 24 * self.V
        relres, iters = ctypes.c_double(), ctypes.c_int()
        rc = self.lib.nd_solve_DNm(self._h, x.data_ptr(), b.data_ptr(), float(prefactor), float(mq), float(tol), int(maxit),
                                   work.data_ptr(), ctypes.byref(relres), ctypes.byref(iters))
        if rc not in (ND_OK, -6):
            self._chk(rc)
        return relres.value, iters.value, rc == ND_OK

    def solve_DNm_mixed(self, ctx32, x, b, prefactor, mq, tol=1e-10, inner_tol=1e-4, max_outer=20, max_inner=500):
        """self: the fp64 context; ctx32: an fp32 context of the same lattice -> (relres, outer, inner_iters, converged)."""
        work64, work32 = self.new_spinor(6), ctx32.new_spinor(10)
        relres, stats = ctypes.c_double(), (_c_int * 2)()
        self.synchronize()
        ctx32.synchronize()
        rc = self.lib.nd_solve_DNm_mixed(self._h, ctx32._h, x.data_ptr(), b.data_ptr(), float(prefactor), float(mq), float(tol),
                                         float(inner_tol), int(max_outer), int(max_inner), work64.data_ptr(),
                                         work32.data_ptr(), ctypes.byref(relres), stats)
        if rc not in (ND_OK, -6):
            self._chk(rc)
        return relres.value, int(stats[0]), int(stats[1]), rc == ND_OK

    def convert_spinor(self, dst, dst_prec, src, src_prec):
        self._chk(self.lib.nd_convert_spinor(self._h, dst.data_ptr(), int(dst_prec), src.data_ptr(), int(src_prec)))

    def lowmodes_compute(self, l, m, tol=1e-8, maxit=50, lextra=8, degree=40, seed=7, l_max=None, stop="residue"):
        """nd_lowmodes_compute with l_min = l, l_max (default l: fixed number of modes), lguard = lextra guard vectors;
        stop = "residue" (rho_k <= tol) or "bound" (bound (2.10) <= tol).
        -> (u [l', 24V] device tensor, nu[l'], resid[l'], stats dict)."""
        l_max = int(l if l_max is None else l_max)
        k = l_max + int(lextra)
        u = self.new_spinor(l_max)
        work = self.new_spinor(int(self.lib.nd_lowmodes_work_spinors(l_max, int(lextra))))
        nu, resid = np.zeros(k), np.zeros(k)
        kappa, bound = np.zeros(2), np.zeros(2)
        lc = ctypes.c_int(0)
        stats = (_c_ll * 2)()
        rule = {"residue": 0, "bound": 1}[stop]
        rc = self.lib.nd_lowmodes_compute(self._h, int(l), l_max, int(lextra), int(degree), float(m), rule, float(tol), int(maxit),
                                          int(seed), u.data_ptr(), nu.ctypes.data_as(_pd), resid.ctypes.data_as(_pd),
                                          ctypes.byref(lc), kappa.ctypes.data_as(_pd), bound.ctypes.data_as(_pd),
                                          work.data_ptr(), stats)
        if rc not in (ND_OK, -6):
            self._chk(rc)
        lp = lc.value
        return u[:lp], nu[:lp].copy(), resid[:lp].copy(), dict(
            iterations=int(stats[0]), stencils=int(stats[1]), converged=(rc == ND_OK), l_chosen=lp, kappa=kappa, bound=bound,
            nu_block=nu, rho_block=resid, nu_guard=nu[lp:].copy(), theta_rest=np.sort(nu[lp:] ** 2),
            message=(self.lib.nd_last_error(self._h).decode() if rc != ND_OK else ""))

    def index_count(self, nvec, zero_tol, degree=8, maxit=40, seed=11):
        """nd_index_count with the sign function set in the context -> (n_plus, n_minus, stats dict with the Ritz values
        `evals` [2, nvec] and residues `resid` [2, nvec] of B_+ and B_-)."""
        nvec = int(nvec)
        work = self.new_spinor(int(self.lib.nd_index_work_spinors(nvec)))
        counts = (_c_int * 2)()
        evals, resid = np.zeros(2 * nvec), np.zeros(2 * nvec)
        stats = (_c_ll * 2)()
        self._chk(self.lib.nd_index_count(self._h, nvec, int(degree), float(zero_tol), int(maxit), int(seed), counts,
                                          evals.ctypes.data_as(_pd), resid.ctypes.data_as(_pd), work.data_ptr(), stats))
        return int(counts[0]), int(counts[1]), dict(evals=evals.reshape(2, nvec), resid=resid.reshape(2, nvec),
                                                    iterations=int(stats[0]), sign_applications=int(stats[1]))

    # -- BLAS-1
    def axpy(self, a, x, y):
        self._chk(self.lib.nd_axpy(self._h, _c2(a), x.data_ptr(), y.data_ptr()))

    def scale(self, a, x):
        self._chk(self.lib.nd_scale(self._h, _c2(a), x.data_ptr()))

    def copy(self, y, x):
        self._chk(self.lib.nd_copy(self._h, y.data_ptr(), x.data_ptr()))

    def dot(self, x, y):
        out = (ctypes.c_double * 2)()
        self._chk(self.lib.nd_dot(self._h, x.data_ptr(), y.data_ptr(), out))
        return complex(out[0], out[1])

    def norm2(self, x):
        out = ctypes.c_double()
        self._chk(self.lib.nd_norm2(self._h, x.data_ptr(), ctypes.byref(out)))
        return out.value

    def gamma5(self, y, x):
        self._chk(self.lib.nd_gamma5(self._h, y.data_ptr(), x.data_ptr()))

    def block_dot(self, v, x):
        l = v.shape[0]
        out = np.zeros(2 * l)
        self._chk(self.lib.nd_block_dot(self._h, l, v.data_ptr(), x.data_ptr(), out.ctypes.data_as(_pd)))
        return out[0::2] + 1j * out[1::2]

    def block_dot_dev(self, v, x, out):
        """out: device float64 tensor of 2l entries, (re, im) pairs; no synchronisation."""
        self._chk(self.lib.nd_block_dot_dev(self._h, v.shape[0], v.data_ptr(), x.data_ptr(), out.data_ptr()))

    def block_axpy_dev(self, a, v, y):
        """a: device float64 tensor of 2l entries, (re, im) pairs; no synchronisation."""
        self._chk(self.lib.nd_block_axpy_dev(self._h, v.shape[0], a.data_ptr(), v.data_ptr(), y.data_ptr()))

    def dot_dev(self, x, y, out):
        self._chk(self.lib.nd_dot_dev(self._h, x.data_ptr(), y.data_ptr(), out.data_ptr()))

    def norm2_dev(self, x, out):
        self._chk(self.lib.nd_norm2_dev(self._h, x.data_ptr(), out.data_ptr()))

    def block_axpy(self, a, v, y):
        a = np.asarray(a, dtype=np.complex128)
        buf = np.empty(2 * len(a))
        buf[0::2], buf[1::2] = a.real, a.imag
        self._chk(self.lib.nd_block_axpy(self._h, len(a), buf.ctypes.data_as(_pd), v.data_ptr(), y.data_ptr()))

    def gaussian(self, x, seed):
        self._chk(self.lib.nd_gaussian(self._h, x.data_ptr(), int(seed)))
