"""ctypes binding of include/tcb200.h and include/tcb200_synth.h.  Same names as the C ABI, marshalling only:
every step of the hot path runs inside libtcb200.so."""
import ctypes
import json
import os

import numpy as np

DOT_NOALLOC_MAX_ELEMS = 536870912          # TCB_DOT_NOALLOC_MAX_ELEMS of include/tcb200.h
TCB_OK, TCB_EINVAL_EXPR, TCB_ESHAPE, TCB_ERANK, TCB_EALIAS, TCB_ENOMEM, TCB_ECUDA, TCB_EUNSUPPORTED, TCB_EINVAL = \
    0, -1, -2, -3, -4, -5, -6, -7, -8

_HERE = os.path.dirname(os.path.abspath(__file__))
_lib = None


class c128(ctypes.Structure):
    _fields_ = [("re", ctypes.c_double), ("im", ctypes.c_double)]


def _c(z):
    z = complex(z)
    return c128(z.real, z.imag)


class kernel_stat(ctypes.Structure):
    _fields_ = [("launches", ctypes.c_int64), ("milliseconds", ctypes.c_double), ("flops", ctypes.c_double),
                ("bytes", ctypes.c_double)]


class TcbError(RuntimeError):
    def __init__(self, code, text):
        super().__init__(f"tcb error {code}: {text}")
        self.code = code


def library_path():
    return os.path.join(_HERE, "libtcb200.so")


# every symbol include/tcb200.h and include/tcb200_synth.h declare
ABI_SYMBOLS = [
    "tcb_ctx_create", "tcb_ctx_destroy", "tcb_ctx_set_option", "tcb_sync", "tcb_last_error", "tcb_strerror",
    "tcb_launch_count", "tcb_tensor_create", "tcb_tensor_alloc", "tcb_tensor_wrap", "tcb_tensor_destroy", "tcb_tensor_info",
    "tcb_tensor_upload", "tcb_tensor_download", "tcb_tensor_fill", "tcb_contract", "tcb_add", "tcb_scale",
    "tcb_denominator_update", "tcb_denominator_divide", "tcb_dot", "tcb_dot_noalloc",
    "tcb_permute", "tcb_permsum", "tcb_antisymmetrize", "tcb_plan_describe", "tcb_measure_fp64_tensor_peak", "tcb_measure_fp64_vector_peak",
    "tcb_capture_begin", "tcb_capture_end", "tcb_graph_launch", "tcb_graph_info", "tcb_graph_destroy",
    "tcb_lane_count", "tcb_lane_set", "tcb_lane_wait", "tcb_pack", "tcb_unpack", "tcb_antisym_pack", "tcb_packed_extent",
    "tcb_timer_start", "tcb_timer_stop", "tcb_kernel_stats", "tcb_kernel_stats_reset", "tcb_plan_describe_host", "tcbx_synth_normal", "tcbx_synth_index_linear",
    "tcbx_synth_mp2_amplitudes",
]


def load_library():
    """Loads libtcb200.so; raises if it has not been built (no fallback of any kind)."""
    global _lib
    if _lib is not None:
        return _lib
    path = library_path()
    if not os.path.exists(path):
        raise TcbError(TCB_ECUDA, f"{path} is missing: run `python -m paper_2409_06759_b200.build` "
                                  "(or __graft_entry__.build()); there is no CPU fallback")
    lib = ctypes.CDLL(path)
    vp, cp, i64p = ctypes.c_void_p, ctypes.c_char_p, ctypes.POINTER(ctypes.c_int64)
    sig = {
        "tcb_ctx_create": [ctypes.POINTER(vp), ctypes.c_int, vp, ctypes.c_size_t],
        "tcb_ctx_destroy": [vp],
        "tcb_ctx_set_option": [vp, cp, cp],
        "tcb_sync": [vp],
        "tcb_tensor_create": [vp, ctypes.POINTER(vp), ctypes.c_int, i64p],
        "tcb_tensor_alloc": [vp, ctypes.POINTER(vp), ctypes.c_int, i64p],
        "tcb_tensor_wrap": [vp, ctypes.POINTER(vp), ctypes.c_int, i64p, vp],
        "tcb_tensor_destroy": [vp],
        "tcb_tensor_info": [vp, ctypes.POINTER(ctypes.c_int), i64p, ctypes.POINTER(vp)],
        "tcb_tensor_upload": [vp, vp, vp],
        "tcb_tensor_download": [vp, vp, vp],
        "tcb_tensor_fill": [vp, vp, c128],
        "tcb_contract": [vp, cp, vp, vp, vp, c128],
        "tcb_add": [vp, cp, vp, vp, c128],
        "tcb_scale": [vp, vp, c128],
        "tcb_denominator_update": [vp, vp, vp, ctypes.POINTER(ctypes.POINTER(ctypes.c_double)), c128],
        "tcb_denominator_divide": [vp, vp, vp, ctypes.POINTER(ctypes.POINTER(ctypes.c_double)), c128],
        "tcb_dot": [vp, vp, vp, vp, ctypes.c_int, c128],
        "tcb_dot_noalloc": [vp, vp, vp, vp, ctypes.c_int, c128],
        "tcb_permute": [vp, cp, vp, vp],
        "tcb_permsum": [vp, vp, vp, ctypes.c_int, ctypes.POINTER(ctypes.c_int32), ctypes.POINTER(c128), c128],
        "tcb_antisymmetrize": [vp, cp, vp, vp, c128],
        "tcb_plan_describe": [vp, cp, vp, vp, vp, ctypes.c_char_p, ctypes.c_size_t],
        "tcb_measure_fp64_tensor_peak": [vp, ctypes.c_double, ctypes.POINTER(ctypes.c_double)],
        "tcb_measure_fp64_vector_peak": [vp, ctypes.c_double, ctypes.POINTER(ctypes.c_double)],
        "tcb_plan_describe_host": [cp, ctypes.c_int, i64p, ctypes.c_int, i64p, ctypes.c_int, i64p, cp, ctypes.c_char_p,
                                   ctypes.c_size_t, i64p, ctypes.c_size_t, i64p, ctypes.c_size_t],
        "tcb_capture_begin": [vp],
        "tcb_capture_end": [vp, ctypes.POINTER(vp)],
        "tcb_graph_launch": [vp, vp],
        "tcb_graph_destroy": [vp],
        "tcb_graph_info": [vp, i64p, i64p, i64p, i64p],
        "tcb_lane_count": [],
        "tcb_pack": [vp, cp, vp, vp],
        "tcb_unpack": [vp, cp, vp, vp, c128],
        "tcb_antisym_pack": [vp, cp, vp, vp, c128],
        "tcb_lane_set": [vp, ctypes.c_int],
        "tcb_lane_wait": [vp, ctypes.c_int, ctypes.c_int],
        "tcb_timer_start": [vp],
        "tcb_kernel_stats": [vp, cp, ctypes.POINTER(kernel_stat)],
        "tcb_kernel_stats_reset": [vp],
        "tcb_timer_stop": [vp, ctypes.POINTER(ctypes.c_double)],
        "tcbx_synth_normal": [vp, vp, ctypes.c_uint64, ctypes.c_uint64, ctypes.c_int, ctypes.POINTER(ctypes.c_int32),
                              ctypes.c_double, ctypes.c_int, i64p, i64p],
        "tcbx_synth_index_linear": [vp, vp],
        "tcbx_synth_mp2_amplitudes": [vp, vp, vp, ctypes.POINTER(ctypes.c_double), ctypes.c_int64,
                                      ctypes.POINTER(ctypes.c_double), ctypes.c_int64],
    }
    for name, args in sig.items():
        fn = getattr(lib, name)
        fn.argtypes = args
        fn.restype = ctypes.c_int
    lib.tcb_last_error.argtypes = [vp]
    lib.tcb_last_error.restype = ctypes.c_char_p
    lib.tcb_strerror.argtypes = [ctypes.c_int]
    lib.tcb_strerror.restype = ctypes.c_char_p
    lib.tcb_packed_extent.argtypes = [ctypes.c_int64, ctypes.c_int]
    lib.tcb_packed_extent.restype = ctypes.c_int64
    lib.tcb_launch_count.argtypes = [vp]
    lib.tcb_launch_count.restype = ctypes.c_int64
    _lib = lib
    return lib


def _ext(extents):
    extents = [int(e) for e in extents]
    return (ctypes.c_int64 * max(len(extents), 1))(*extents), len(extents)


def plan_describe_host(expr, ext_d, ext_l, ext_r, options=None, want_tables=False):
    """Host-only planner (no device needed).  Returns the plan dict, and (offM, offN) if want_tables."""
    lib = load_library()
    ed, rd = _ext(ext_d)
    el, rl = _ext(ext_l)
    er, rr = _ext(ext_r)
    buf = ctypes.create_string_buffer(2048)
    opt = options.encode() if options else None
    rc = lib.tcb_plan_describe_host(expr.encode(), rd, ed, rl, el, rr, er, opt, buf, 2048, None, 0, None, 0)
    if rc != 0:
        raise TcbError(rc, lib.tcb_strerror(rc).decode() + ": " + buf.value.decode())
    plan = json.loads(buf.value.decode())
    if not want_tables:
        return plan
    offM = np.zeros(plan["M"], dtype=np.int64)
    offN = np.zeros(plan["N"], dtype=np.int64)
    i64p = ctypes.POINTER(ctypes.c_int64)
    rc = lib.tcb_plan_describe_host(expr.encode(), rd, ed, rl, el, rr, er, opt, buf, 2048,
                                    offM.ctypes.data_as(i64p), offM.size, offN.ctypes.data_as(i64p), offN.size)
    if rc != 0:
        raise TcbError(rc, lib.tcb_strerror(rc).decode())
    return plan, offM, offN


class Tensor:
    """Handle of a device tensor (tcb_tensor).  Column-major: the first index has unit stride."""

    def __init__(self, ctx, handle, extents, keepalive=None):
        self.ctx, self.handle, self.extents, self._keep = ctx, handle, tuple(int(e) for e in extents), keepalive

    @property
    def size(self):
        return int(np.prod(self.extents)) if self.extents else 1

    @property
    def nbytes(self):
        return self.size * 16

    def destroy(self):
        # a tensor must not outlive its context: after Context.destroy() the handle is already gone
        if self.handle is not None and self.ctx.handle is not None:
            self.ctx.lib.tcb_tensor_destroy(self.handle)
        self.handle = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


class Context:
    """tcb_ctx.  Method names follow the C ABI (tcb_ prefix dropped)."""

    def __init__(self, device=0, stream=None, workspace_bytes=0):
        self.lib = load_library()
        h = ctypes.c_void_p()
        rc = self.lib.tcb_ctx_create(ctypes.byref(h), int(device), stream, int(workspace_bytes))
        if rc != 0:
            raise TcbError(rc, self.lib.tcb_strerror(rc).decode() +
                           " (tcb_ctx_create: a CUDA device is required, there is no CPU fallback)")
        self.handle = h
        self._tensors = []

    def _check(self, rc):
        if rc != 0:
            raise TcbError(rc, f"{self.lib.tcb_strerror(rc).decode()}: {self.lib.tcb_last_error(self.handle).decode()}")

    def destroy(self):
        """Destroys every tensor still alive on this context, then the context."""
        if getattr(self, "handle", None) is not None:
            for ref in list(self._tensors):
                t = ref()
                if t is not None:
                    t.destroy()
            self._tensors.clear()
            self.lib.tcb_ctx_destroy(self.handle)
            self.handle = None

    def _track(self, t):
        import weakref
        self._tensors.append(weakref.ref(t))
        if len(self._tensors) > 4096:
            self._tensors = [r for r in self._tensors if r() is not None and r().handle is not None]
        return t

    def set_option(self, key, value):
        self._check(self.lib.tcb_ctx_set_option(self.handle, key.encode(), str(value).encode()))

    def sync(self):
        self._check(self.lib.tcb_sync(self.handle))

    def launch_count(self):
        return int(self.lib.tcb_launch_count(self.handle))

    # ---- tensors ----
    def tensor_create(self, extents, zero=True):
        """zero=False: tcb_tensor_alloc, contents undefined until written (for targets of '=' operations)"""
        e, r = _ext(extents)
        h = ctypes.c_void_p()
        fn = self.lib.tcb_tensor_create if zero else self.lib.tcb_tensor_alloc
        self._check(fn(self.handle, ctypes.byref(h), r, e))
        return self._track(Tensor(self, h, extents))

    def tensor_wrap(self, extents, device_ptr, keepalive=None):
        e, r = _ext(extents)
        h = ctypes.c_void_p()
        self._check(self.lib.tcb_tensor_wrap(self.handle, ctypes.byref(h), r, e, ctypes.c_void_p(int(device_ptr))))
        return self._track(Tensor(self, h, extents, keepalive))

    def tensor_wrap_torch(self, t, extents):
        """Borrow a torch CUDA complex128 buffer (plumbing only: torch owns the memory)."""
        assert t.is_cuda and t.is_contiguous() and t.element_size() == 16 and t.numel() == int(np.prod(extents))
        return self.tensor_wrap(extents, t.data_ptr(), keepalive=t)

    def tensor_upload(self, t, host):
        host = np.asarray(host, dtype=np.complex128)
        assert host.shape == t.extents, (host.shape, t.extents)
        host = np.asfortranarray(host)
        self._check(self.lib.tcb_tensor_upload(self.handle, t.handle, host.ctypes.data_as(ctypes.c_void_p)))
        self.sync()            # `host` may be a temporary
        return t

    def tensor_upload_raw(self, t, host_ptr):
        """host_ptr: address of a (pinned) host buffer in the tensor's layout; stream-ordered, no sync."""
        self._check(self.lib.tcb_tensor_upload(self.handle, t.handle, ctypes.c_void_p(int(host_ptr))))

    def tensor_download_raw(self, t, host_ptr):
        self._check(self.lib.tcb_tensor_download(self.handle, t.handle, ctypes.c_void_p(int(host_ptr))))

    def tensor_from_numpy(self, host):
        host = np.asarray(host, dtype=np.complex128)
        return self.tensor_upload(self.tensor_create(host.shape), host)

    def tensor_download(self, t):
        out = np.empty(t.extents, dtype=np.complex128, order="F")
        self._check(self.lib.tcb_tensor_download(self.handle, t.handle, out.ctypes.data_as(ctypes.c_void_p)))
        return out

    def tensor_device_ptr(self, t):
        """Device address of the tensor's storage (tcb_tensor_info)."""
        ptr = ctypes.c_void_p()
        self._check(self.lib.tcb_tensor_info(t.handle, None, None, ctypes.byref(ptr)))
        return ptr.value

    def tensor_fill(self, t, value):
        self._check(self.lib.tcb_tensor_fill(self.handle, t.handle, _c(value)))

    # ---- hot path ----
    def contract(self, expr, D, L, R, alpha=1.0):
        self._check(self.lib.tcb_contract(self.handle, expr.encode(), D.handle, L.handle, R.handle, _c(alpha)))

    def add(self, expr, D, L, alpha=1.0):
        self._check(self.lib.tcb_add(self.handle, expr.encode(), D.handle, L.handle, _c(alpha)))

    def scale(self, D, alpha):
        self._check(self.lib.tcb_scale(self.handle, D.handle, _c(alpha)))

    def _denominator(self, fn, T, R, eps, alpha):
        import numpy as np
        keep = [None if e is None else np.ascontiguousarray(e, dtype=np.float64) for e in eps]
        dp = ctypes.POINTER(ctypes.c_double)
        arr = (dp * len(keep))(*[ctypes.cast(None, dp) if e is None else e.ctypes.data_as(dp) for e in keep])
        self._check(fn(self.handle, T.handle, R.handle, arr, _c(alpha)))

    def denominator_update(self, T, R, eps, alpha=1.0):
        """T[i0,i1,..] += alpha * R[i0,i1,..] / (eps[0][i0] + eps[1][i1] + ...); eps: one real vector (or None) per index."""
        self._denominator(self.lib.tcb_denominator_update, T, R, eps, alpha)

    def denominator_divide(self, T, R, eps, alpha=1.0):
        """T[i0,i1,..] = alpha * R[i0,i1,..] / (eps[0][i0] + eps[1][i1] + ...); T is not read."""
        self._denominator(self.lib.tcb_denominator_divide, T, R, eps, alpha)

    def dot(self, D, X, Y, conjugate_x=True, alpha=1.0):
        """D (rank 0) = alpha * sum conj?(X) * Y"""
        self._check(self.lib.tcb_dot(self.handle, D.handle, X.handle, Y.handle, int(bool(conjugate_x)), _c(alpha)))

    def dot_noalloc(self, D, X, Y, conjugate_x=True, alpha=1.0):
        """tcb_dot with its scratch in a fixed device array inside the library: no allocation of any kind; at most
        DOT_NOALLOC_MAX_ELEMS elements; calls that overlap on the GPU race on the array"""
        self._check(self.lib.tcb_dot_noalloc(self.handle, D.handle, X.handle, Y.handle, int(bool(conjugate_x)), _c(alpha)))

    def permute(self, expr, D, L):
        self._check(self.lib.tcb_permute(self.handle, expr.encode(), D.handle, L.handle))

    def permsum(self, D, X, perms, coefs, beta=1.0):
        perms = np.ascontiguousarray(np.asarray(perms, dtype=np.int32).reshape(-1))
        n = len(coefs)
        cf = (c128 * n)(*[_c(c) for c in coefs])
        self._check(self.lib.tcb_permsum(self.handle, D.handle, X.handle, n,
                                         perms.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)), cf, _c(beta)))

    def antisymmetrize(self, spec, D, X, alpha=1.0):
        self._check(self.lib.tcb_antisymmetrize(self.handle, spec.encode(), D.handle, X.handle, _c(alpha)))

    def pack(self, spec, D, L):
        """'Vp(a<b,c<d)=V(a,b,c,d)': antisymmetric index groups stored as one packed index each (tcb_pack)"""
        self._check(self.lib.tcb_pack(self.handle, spec.encode(), D.handle, L.handle))

    def unpack(self, spec, D, L, alpha=1.0):
        """'R(a,b,i,j)+=Rp(a<b,i<j)': D (+)= alpha * sign * Lp[packed position] (tcb_unpack)"""
        self._check(self.lib.tcb_unpack(self.handle, spec.encode(), D.handle, L.handle, _c(alpha)))

    def antisym_pack(self, spec, D, L, alpha=1.0):
        """'R(a<b<c,i<j<k)+=X(a,i,b<c,j<k)': P(a/bc)P(i/jk) on packed storage, D (+)= alpha * signed sum over the shuffles
        (tcb_antisym_pack)"""
        self._check(self.lib.tcb_antisym_pack(self.handle, spec.encode(), D.handle, L.handle, _c(alpha)))

    def packed_extent(self, n, k):
        return int(self.lib.tcb_packed_extent(int(n), int(k)))

    def plan_describe(self, expr, D, L, R):
        buf = ctypes.create_string_buffer(2048)
        self._check(self.lib.tcb_plan_describe(self.handle, expr.encode(), D.handle, L.handle, R.handle, buf, 2048))
        return json.loads(buf.value.decode())

    # ---- measurement ----
    def measure_fp64_tensor_peak(self, milliseconds=200.0):
        out = ctypes.c_double()
        self._check(self.lib.tcb_measure_fp64_tensor_peak(self.handle, float(milliseconds), ctypes.byref(out)))
        return out.value

    def measure_fp64_vector_peak(self, milliseconds=200.0):
        out = ctypes.c_double()
        self._check(self.lib.tcb_measure_fp64_vector_peak(self.handle, float(milliseconds), ctypes.byref(out)))
        return out.value

    def kernel_stats(self, kernel):
        out = kernel_stat()
        self._check(self.lib.tcb_kernel_stats(self.handle, kernel.encode(), ctypes.byref(out)))
        return {"launches": int(out.launches), "ms": out.milliseconds, "flops": out.flops, "bytes": out.bytes}

    def kernel_stats_reset(self):
        self._check(self.lib.tcb_kernel_stats_reset(self.handle))

    def capture_begin(self):
        self._check(self.lib.tcb_capture_begin(self.handle))

    def capture_end(self):
        """Returns an opaque graph handle for graph_launch / graph_destroy."""
        g = ctypes.c_void_p()
        self._check(self.lib.tcb_capture_end(self.handle, ctypes.byref(g)))
        return g

    def graph_launch(self, g):
        self._check(self.lib.tcb_graph_launch(self.handle, g))

    def graph_info(self, g):
        """{'nodes', 'edges', 'launches'} of a captured graph"""
        n, e, k, d = ctypes.c_int64(), ctypes.c_int64(), ctypes.c_int64(), ctypes.c_int64()
        self._check(self.lib.tcb_graph_info(g, ctypes.byref(n), ctypes.byref(e), ctypes.byref(k), ctypes.byref(d)))
        return {"nodes": n.value, "edges": e.value, "launches": k.value, "depth": d.value}

    def lane_count(self):
        return int(self.lib.tcb_lane_count())

    def lane_set(self, lane):
        self._check(self.lib.tcb_lane_set(self.handle, int(lane)))

    def lane_wait(self, lane, on_lane):
        self._check(self.lib.tcb_lane_wait(self.handle, int(lane), int(on_lane)))

    def graph_destroy(self, g):
        self.lib.tcb_graph_destroy(g)

    def timer_start(self):
        self._check(self.lib.tcb_timer_start(self.handle))

    def timer_stop(self):
        out = ctypes.c_double()
        self._check(self.lib.tcb_timer_stop(self.handle, ctypes.byref(out)))
        return out.value

    # ---- device-side synthetic inputs (include/tcb200_synth.h) ----
    def synth_normal(self, t, seed, tensor_id, antisym=(), sigma=1.0, hermitian=False, label_offset=None,
                     label_extents=None):
        pairs = [int(x) for p in antisym for x in p]
        pa = (ctypes.c_int32 * max(len(pairs), 1))(*pairs)
        lo = _ext(label_offset)[0] if label_offset is not None else None
        le = _ext(label_extents)[0] if label_extents is not None else None
        self._check(self.lib.tcbx_synth_normal(self.handle, t.handle, int(seed), int(tensor_id), len(antisym), pa,
                                               float(sigma), 1 if hermitian else 0, lo, le))

    def synth_index_linear(self, t):
        self._check(self.lib.tcbx_synth_index_linear(self.handle, t.handle))

    def synth_mp2_amplitudes(self, T, vvoo, eo, ev):
        eo = np.ascontiguousarray(eo, dtype=np.float64)
        ev = np.ascontiguousarray(ev, dtype=np.float64)
        dp = ctypes.POINTER(ctypes.c_double)
        self._check(self.lib.tcbx_synth_mp2_amplitudes(self.handle, T.handle, vvoo.handle, eo.ctypes.data_as(dp),
                                                       len(eo), ev.ctypes.data_as(dp), len(ev)))
        self.sync()
