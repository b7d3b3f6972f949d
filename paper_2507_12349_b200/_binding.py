"""ctypes marshalling for include/cos.h.  Same function names as the C-ABI.

Device arrays are torch CUDA tensors (PyTorch is used for device memory and streams only); the
binding passes their data pointers and the current CUDA stream.  A missing shared library raises
ImportError-like CosError loudly: there is no Python / CPU implementation behind these calls.
"""
import ctypes
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
# COS_B200_LIB selects another build of the same library (the self-check build of tests/test_gpu_selfcheck.py)
_LIB_PATH = os.environ.get("COS_B200_LIB") or os.path.join(_HERE, "libcos_b200.so")
_lib = None

COS_OK, COS_EINVAL, COS_ENOMEM, COS_ECUDA, COS_EUNSUPPORTED = 0, 1, 2, 3, 4
COS_LATTICE_SQUARE, COS_LATTICE_HONEYCOMB = 0, 1
COS_BUILD_HOST_ONLY, COS_BUILD_NO_FUSED, COS_BUILD_UNIFORM_SHIFT = 1, 2, 4
COS_DET_FP64, COS_DET_DD = 0, 1
COS_DET_STATIC_SCRATCH_BYTES = 16 << 20
TUNE = {"prefetch": 0, "warps_per_cta": 1, "blocks_per_cta_cap": 2, "pdl": 3, "fused": 4, "host_slices": 5,
        "tiles_per_chunk": 6}

INFO = {
    "n_layers": 0, "n_states": 1, "n_edges": 2, "n_readout_edges": 3, "n_out": 4, "max_layer_states": 5,
    "n_masks": 6, "n_rows": 7, "n_fma": 8, "program_bytes": 9, "d": 10, "n_blocks": 11,
    "n_states_unpruned": 12, "workspace_bytes": 13, "n_launches": 14, "order_mask": 15, "reserved_batch": 16,
    "device": 19, "fused": 20,
    "layer_states": 100, "layer_edges": 200, "layer_masks": 300,
}

EXPORTS = [
    "cos_build", "cos_build_ex", "cos_eval", "cos_free", "cos_set_workspace_limit", "cos_info",
    "cos_last_error", "cos_tab_build", "cos_tabulate", "cos_tab_free", "cos_measure_fp64_fma_peak",
    "cos_eval_host", "cos_set_profiling", "cos_get_layer_times", "cos_build_orders", "cos_flux_weights",
    "cos_det_workspace_bytes", "cos_det_eval", "cos_reserve", "cos_set_tuning", "cos_debug_check_failures",
    "cos_equivalence_stats", "cos_det_eval_static",
]


class CosError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("cos error %d: %s" % (code, msg))
        self.code = code


def lib_path():
    return _LIB_PATH


def load_library():
    """dlopen libcos_b200.so (built by `python -m paper_2507_12349_b200.build` / __graft_entry__.build())."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise CosError(COS_ECUDA, "libcos_b200.so is missing at %s: build it with "
                       "`python -m paper_2507_12349_b200.build` (there is no fallback implementation)" % _LIB_PATH)
    lib = ctypes.CDLL(_LIB_PATH)
    vp, ip, dp, llp = ctypes.c_void_p, ctypes.c_int, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_longlong)
    lib.cos_build.restype = ctypes.c_int
    lib.cos_build.argtypes = [ip, ip, ip, dp, ip, ctypes.POINTER(vp)]
    lib.cos_build_ex.restype = ctypes.c_int
    lib.cos_build_ex.argtypes = [ip, ip, ip, dp, ip, ip, ctypes.POINTER(vp)]
    lib.cos_eval.restype = ctypes.c_int
    lib.cos_eval.argtypes = [vp, vp, ctypes.c_longlong, vp, vp]
    lib.cos_free.restype = None
    lib.cos_free.argtypes = [vp]
    lib.cos_set_workspace_limit.restype = ctypes.c_int
    lib.cos_set_workspace_limit.argtypes = [vp, ctypes.c_longlong]
    lib.cos_info.restype = ctypes.c_int
    lib.cos_info.argtypes = [vp, ip, llp]
    lib.cos_last_error.restype = ctypes.c_char_p
    lib.cos_last_error.argtypes = []
    lib.cos_tab_build.restype = ctypes.c_int
    lib.cos_tab_build.argtypes = [ip, ip, ip, ctypes.c_double, ip, vp, ctypes.POINTER(vp)]
    lib.cos_tabulate.restype = ctypes.c_int
    lib.cos_tabulate.argtypes = [vp, ip, vp, vp, ctypes.c_longlong, vp, vp]
    lib.cos_tab_free.restype = None
    lib.cos_tab_free.argtypes = [vp]
    lib.cos_eval_host.restype = ctypes.c_int
    lib.cos_eval_host.argtypes = [vp, vp, vp, vp, ctypes.c_longlong, vp, vp]
    lib.cos_set_profiling.restype = ctypes.c_int
    lib.cos_set_profiling.argtypes = [vp, ip]
    lib.cos_get_layer_times.restype = ctypes.c_int
    lib.cos_get_layer_times.argtypes = [vp, ip, dp, llp]
    lib.cos_build_orders.restype = ctypes.c_int
    lib.cos_build_orders.argtypes = [ip, ip, ip, dp, ctypes.c_uint, ip, ctypes.POINTER(vp)]
    lib.cos_flux_weights.restype = ctypes.c_int
    lib.cos_flux_weights.argtypes = [ip, ctypes.c_uint, dp, vp, vp, ctypes.c_longlong, vp, vp, vp]
    lib.cos_det_workspace_bytes.restype = ctypes.c_longlong
    lib.cos_det_workspace_bytes.argtypes = [ip, ip, ip, ctypes.c_longlong]
    lib.cos_det_eval.restype = ctypes.c_int
    lib.cos_det_eval.argtypes = [ip, ip, ip, ip, dp, ip, vp, ctypes.c_longlong, vp, vp, ctypes.c_longlong, vp]
    lib.cos_det_eval_static.restype = ctypes.c_int
    lib.cos_det_eval_static.argtypes = [ip, ip, ip, ip, dp, ip, vp, ctypes.c_longlong, vp, vp]
    lib.cos_measure_fp64_fma_peak.restype = ctypes.c_int
    lib.cos_measure_fp64_fma_peak.argtypes = [dp]
    lib.cos_equivalence_stats.restype = ctypes.c_int
    lib.cos_equivalence_stats.argtypes = [ip, ip, ip, dp, ip, ip, llp]
    lib.cos_debug_check_failures.restype = ctypes.c_int
    lib.cos_debug_check_failures.argtypes = [llp, llp]
    lib.cos_reserve.restype = ctypes.c_int
    lib.cos_reserve.argtypes = [vp, ctypes.c_longlong]
    lib.cos_set_tuning.restype = ctypes.c_int
    lib.cos_set_tuning.argtypes = [vp, ip, ctypes.c_longlong]
    _lib = lib
    return lib


def cos_last_error():
    return load_library().cos_last_error().decode("utf-8", "replace")


def _check(rc):
    if rc != COS_OK:
        raise CosError(rc, cos_last_error())


def _shifts_arg(shifts):
    if shifts is None:
        return None, None
    arr = (ctypes.c_double * len(shifts))(*[float(s) for s in shifts])
    return arr, ctypes.cast(arr, ctypes.POINTER(ctypes.c_double))


def cos_build_ex(n, n_flavors, lattice, shifts, readout_envelope, flags=0):
    """-> opaque handle (int).  shifts: None (uniform CoS), a sequence of n_flavors sigma values (SB-CoS), or one value
    with COS_BUILD_UNIFORM_SHIFT in flags (uniform CoS with a counterterm)."""
    lib = load_library()
    keep, p = _shifts_arg(shifts)
    h = ctypes.c_void_p()
    _check(lib.cos_build_ex(int(n), int(n_flavors), int(lattice), p, int(readout_envelope), int(flags), ctypes.byref(h)))
    _shape_cache.pop(h.value, None)               # a new handle may reuse the address of one freed outside the binding
    return h.value


def cos_build_orders(n, n_flavors, lattice, shifts, order_mask, flags=0):
    """All-subset layout restricted to the allowed orders: bit k of order_mask <-> subsets with |S| = k."""
    lib = load_library()
    keep, p = _shifts_arg(shifts)
    h = ctypes.c_void_p()
    _check(lib.cos_build_orders(int(n), int(n_flavors), int(lattice), p, int(order_mask), int(flags), ctypes.byref(h)))
    _shape_cache.pop(h.value, None)               # a new handle may reuse the address of one freed outside the binding
    return h.value


def cos_flux_weights(n, order_mask, lambdas, C_dev, Q_dev, batch, W_dev, Phi_dev=None, stream=None):
    """W[c] = sum_{|S| in U} |lambda_|S| C_S Q_S| / binom(n, |S|) (Eq. 6-7).  lambdas: n+1 floats (index = order);
    C_dev / Q_dev / Phi_dev: torch.float64 CUDA tensors [2^n-1, batch] (Q_dev, Phi_dev may be None); W_dev: [batch]."""
    lam = (ctypes.c_double * (int(n) + 1))(*[float(x) for x in lambdas])
    _check(load_library().cos_flux_weights(
        int(n), int(order_mask), ctypes.cast(lam, ctypes.POINTER(ctypes.c_double)),
        _dev_ptr(C_dev, "torch.float64", ((1 << int(n)) - 1) * int(batch), "C_dev"),
        None if Q_dev is None else _dev_ptr(Q_dev, "torch.float64", ((1 << int(n)) - 1) * int(batch), "Q_dev"), int(batch),
        _dev_ptr(W_dev, "torch.float64", int(batch), "W_dev"),
        None if Phi_dev is None else _dev_ptr(Phi_dev, "torch.float64", ((1 << int(n)) - 1) * int(batch), "Phi_dev"),
        _stream_ptr(stream)))


def cos_det_workspace_bytes(n, n_blocks, precision, batch):
    """Bytes of device scratch cos_det_eval needs (-1 on bad arguments)."""
    return int(load_library().cos_det_workspace_bytes(int(n), int(n_blocks), int(precision), int(batch)))


def cos_det_eval(n, n_flavors, n_blocks, shifts, precision, G_dev, batch, out_dev, work_dev, stream=None,
                 lattice=COS_LATTICE_SQUARE):
    """Determinant-polynomial route (Eq. 34-38): all 2^n-1 connected values of every configuration.
    precision: COS_DET_FP64 or COS_DET_DD (double-double).  G_dev: torch.float64 CUDA [n_blocks*d*d, batch], d = n (square)
    or 2n (lattice=COS_LATTICE_HONEYCOMB: sublattice-summed, Eq. 54-55);
    out_dev: [2^n-1, batch]; work_dev: any contiguous CUDA tensor of at least
    cos_det_workspace_bytes(n, n_blocks, precision, batch) bytes (torch allocations are suitably aligned)."""
    keep, p = _shifts_arg(shifts)
    if not work_dev.is_cuda or not work_dev.is_contiguous():
        raise ValueError("work_dev must be a contiguous CUDA tensor")
    d = int(n) * (2 if int(lattice) == COS_LATTICE_HONEYCOMB else 1)
    _check(load_library().cos_det_eval(
        int(n), int(n_flavors), int(n_blocks), int(lattice), p, int(precision),
        _dev_ptr(G_dev, "torch.float64", int(n_blocks) * d * d * int(batch), "G_dev"), int(batch),
        _dev_ptr(out_dev, "torch.float64", ((1 << int(n)) - 1) * int(batch), "out_dev"), work_dev.data_ptr(),
        int(work_dev.numel() * work_dev.element_size()), _stream_ptr(stream)))


def cos_det_eval_static(n, n_flavors, n_blocks, shifts, precision, G_dev, batch, out_dev, stream=None,
                        lattice=COS_LATTICE_SQUARE):
    """cos_det_eval without a work buffer, for code that is not allowed to allocate device memory (a sampler loop that
    must not stall the GPU on cudaMalloc, a plug-in inside a program whose own pool already owns all of HBM, a
    latency-bounded service): the scratch is a 16 MiB array built into libcos_b200.so, so no call allocates anything.
    Same arguments and bit-identical results as cos_det_eval; problems whose cos_det_workspace_bytes(...) exceeds
    COS_DET_STATIC_SCRATCH_BYTES raise CosError(COS_EUNSUPPORTED).  All calls on a device share the one array: keep them
    on one stream (overlapping calls race), and make the first call on each device during initialisation, before any
    stream capture -- it looks up the array's device address.  See include/cos.h."""
    keep, p = _shifts_arg(shifts)
    d = int(n) * (2 if int(lattice) == COS_LATTICE_HONEYCOMB else 1)
    _check(load_library().cos_det_eval_static(
        int(n), int(n_flavors), int(n_blocks), int(lattice), p, int(precision),
        _dev_ptr(G_dev, "torch.float64", int(n_blocks) * d * d * int(batch), "G_dev"), int(batch),
        _dev_ptr(out_dev, "torch.float64", ((1 << int(n)) - 1) * int(batch), "out_dev"), _stream_ptr(stream)))


def cos_build(n, n_flavors, lattice, shifts, readout_envelope):
    return cos_build_ex(n, n_flavors, lattice, shifts, readout_envelope, 0)


def _stream_ptr(stream):
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    return getattr(stream, "cuda_stream", stream)


def _dev_ptr(t, dtype_name, numel=0, what="tensor"):
    """Data pointer of a contiguous CUDA tensor of the given dtype holding at least `numel` elements."""
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.is_contiguous() and str(t.dtype) == dtype_name):
        raise CosError(COS_EINVAL, "%s: expected a contiguous CUDA tensor of dtype %s" % (what, dtype_name))
    if t.numel() < numel:
        raise CosError(COS_EINVAL, "%s: %d elements, the call needs %d" % (what, t.numel(), numel))
    return t.data_ptr()


def cos_eval(handle, G_dev, batch, out_dev, stream=None):
    """G_dev: torch.float64 CUDA tensor [n_blocks*d*d, batch] (batch contiguous); out_dev: [n_out, batch]."""
    lib = load_library()
    B, sh = int(batch), _shape(handle)
    d = sh["d"]
    _check(lib.cos_eval(handle, _dev_ptr(G_dev, "torch.float64", sh["n_blocks"] * d * d * B, "G_dev"), B,
                        _dev_ptr(out_dev, "torch.float64", sh["n_out"] * B, "out_dev"),
                        _stream_ptr(stream)))


def cos_reserve(handle, batch):
    """Allocate the layer-slab workspace for batches up to `batch` now, so that cos_eval only enqueues kernels."""
    _check(load_library().cos_reserve(handle, int(batch)))


def cos_set_tuning(handle, what, value):
    """what: a key of TUNE ("prefetch", "warps_per_cta", "blocks_per_cta_cap", "pdl", "fused", "host_slices",
    "tiles_per_chunk") or its integer code."""
    code = TUNE[what] if isinstance(what, str) else int(what)
    _check(load_library().cos_set_tuning(handle, code, int(value)))


# constants of a handle that the size checks of cos_eval / cos_eval_host need on every call: fetched once per handle
# (three cos_info round trips otherwise sit inside the timed step of launch-bound workloads), dropped by cos_free
_shape_cache = {}


def _shape(handle):
    s = _shape_cache.get(handle)
    if s is None:
        s = {k: cos_info(handle, k) for k in ("d", "n_blocks", "n_out", "n_layers")}
        _shape_cache[handle] = s
    return s


def cos_free(handle):
    _shape_cache.pop(handle, None)
    load_library().cos_free(handle)


def cos_set_workspace_limit(handle, nbytes):
    _check(load_library().cos_set_workspace_limit(handle, int(nbytes)))


def cos_info(handle, what, layer=0):
    code = INFO[what] if isinstance(what, str) else int(what)
    if code >= 100:
        code += int(layer)
    v = ctypes.c_longlong(0)
    _check(load_library().cos_info(handle, code, ctypes.byref(v)))
    return v.value


def cos_tab_build(lattice, L, n_blocks, beta, n_tau, table_host):
    """table_host: C-contiguous numpy float64 [n_blocks][n_sub^2][L*L][n_tau]."""
    import numpy as np
    t = np.ascontiguousarray(table_host, dtype=np.float64)
    tab = ctypes.c_void_p()
    _check(load_library().cos_tab_build(int(lattice), int(L), int(n_blocks), float(beta), int(n_tau),
                                        t.ctypes.data, ctypes.byref(tab)))
    return tab.value


def cos_tabulate(tab, n, sites_dev, tau_dev, batch, G_dev, stream=None):
    """sites_dev int32 [n,2,batch], tau_dev fp64 [n,batch], G_dev fp64 [n_blocks*d*d, batch] (at least n*n*batch: the
    library knows the table's block and sublattice counts, the binding checks the part it can)."""
    n, B = int(n), int(batch)
    _check(load_library().cos_tabulate(tab, n, _dev_ptr(sites_dev, "torch.int32", n * 2 * B, "sites_dev"),
                                       _dev_ptr(tau_dev, "torch.float64", n * B, "tau_dev"), B,
                                       _dev_ptr(G_dev, "torch.float64", n * n * B, "G_dev"), _stream_ptr(stream)))


def _host_ptr(t, dtype_name, numel=0, what="tensor"):
    import torch
    if not (isinstance(t, torch.Tensor) and not t.is_cuda and t.is_contiguous() and str(t.dtype) == dtype_name):
        raise CosError(COS_EINVAL, "%s: expected a contiguous host tensor of dtype %s" % (what, dtype_name))
    if t.numel() < numel:
        raise CosError(COS_EINVAL, "%s: %d elements, the call needs %d" % (what, t.numel(), numel))
    return t.data_ptr()


def cos_eval_host(handle, tab, sites_host, tau_host, batch, out_host, stream=None):
    """Host-buffer pipeline: sites_host int32 [n,2,batch], tau_host fp64 [n,batch], out_host fp64 [n_out,batch]
    (torch CPU tensors, ideally pinned).  Synchronises the stream before returning."""
    B = int(batch)
    sh = _shape(handle)
    n = sh["n_layers"] // 2
    _check(load_library().cos_eval_host(handle, tab, _host_ptr(sites_host, "torch.int32", n * 2 * B, "sites_host"),
                                        _host_ptr(tau_host, "torch.float64", n * B, "tau_host"), B,
                                        _host_ptr(out_host, "torch.float64", sh["n_out"] * B, "out_host"),
                                        _stream_ptr(stream)))


def cos_set_profiling(handle, on):
    _check(load_library().cos_set_profiling(handle, int(bool(on))))


def cos_get_layer_times(handle):
    """-> (list of per-layer milliseconds accumulated since the last call, number of profiled cos_eval calls)."""
    nl = cos_info(handle, "n_layers")
    ms = (ctypes.c_double * nl)()
    n = ctypes.c_longlong(0)
    _check(load_library().cos_get_layer_times(handle, nl, ms, ctypes.byref(n)))
    return list(ms), n.value


def cos_tab_free(tab):
    load_library().cos_tab_free(tab)


def cos_equivalence_stats(n, n_flavors, lattice, shifts, readout_envelope, flags=0):
    """Future / past equivalence classes of the compiled DAG (Eq. 25-28), host only.
    -> dict(states, edges, future_classes, edges_after_future_merge, past_classes, edges_after_past_merge)."""
    keep, p = _shifts_arg(shifts)
    out = (ctypes.c_longlong * 6)()
    _check(load_library().cos_equivalence_stats(int(n), int(n_flavors), int(lattice), p, int(readout_envelope), int(flags), out))
    return dict(zip(("states", "edges", "future_classes", "edges_after_future_merge", "past_classes",
                     "edges_after_past_merge"), [int(x) for x in out]))


def cos_debug_check_failures():
    """-> (total, [8 counters by kind]); total = -1 for a library built without COS_CHECK_BOUNDS."""
    total = ctypes.c_longlong(0)
    kinds = (ctypes.c_longlong * 8)()
    _check(load_library().cos_debug_check_failures(ctypes.byref(total), kinds))
    return total.value, list(kinds)


def cos_measure_fp64_fma_peak():
    v = ctypes.c_double(0.0)
    _check(load_library().cos_measure_fp64_fma_peak(ctypes.byref(v)))
    return v.value


def dag_summary(handle):
    """Convenience: the cos_info counters as a dict (host data only)."""
    keys = ["n_layers", "n_states", "n_edges", "n_readout_edges", "n_out", "max_layer_states", "n_masks",
            "n_rows", "n_fma", "program_bytes", "d", "n_blocks", "n_states_unpruned", "order_mask"]
    out = {k: cos_info(handle, k) for k in keys}
    nl = out["n_layers"]
    out["layer_states"] = [cos_info(handle, "layer_states", l) for l in range(nl)]
    out["layer_edges"] = [cos_info(handle, "layer_edges", l) for l in range(nl)]
    out["layer_masks"] = [cos_info(handle, "layer_masks", l) for l in range(nl)]
    return out
