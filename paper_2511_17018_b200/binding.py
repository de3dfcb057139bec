"""ctypes binding of libtpcclus.so -- argument marshalling only.

Module-level functions carry the names of the C ABI (include/tpcclus.h):
``tpcclus_workspace_bytes``, ``tpcclus_create``, ``tpcclus_run``, ``tpcclus_run_host``,
``tpcclus_destroy`` ...  ``Clusterizer`` bundles them with the torch tensors that own the
device memory (workspace, clusters, counters).  Nothing here computes: every step of the
path runs in the CUDA kernels behind ``tpcclus_run``.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libtpcclus.so")

MODE_FAST, MODE_DETERMINISTIC = 0, 1
RTC = 1
COG_GATED = 2
COG_SHARED = 4
STATUS_OVERFLOW, STATUS_BAD_DIGITS, STATUS_NO_PACKED, STATUS_INTERNAL = 1, 2, 4, 0x80000000
FLAG_EDGE_PAD, FLAG_EDGE_TIME, FLAG_SATURATED = 1, 2, 4

# include/tpcclus.h: tpcclus_digit (8 B) and tpcclus_cluster (32 B)
DIGIT_DTYPE = np.dtype([("charge", "<u2"), ("time", "<u2"), ("pad", "u1"), ("row", "u1"), ("sector", "u1"),
                        ("reserved", "u1")])
CLUSTER_DTYPE = np.dtype([("pad_mean", "<f4"), ("time_mean", "<f4"), ("sigma_pad", "<f4"), ("sigma_time", "<f4"),
                          ("q_tot", "<u4"), ("q_max", "<u2"), ("time_peak", "<u2"), ("pad_peak", "u1"),
                          ("row", "u1"), ("sector", "u1"), ("flags", "u1"), ("reserved", "<u4")])
CLUSTER16_DTYPE = np.dtype([("time_fix_pad_peak", "<u4"), ("pad_fix", "<u2"), ("time_peak", "<u2"), ("q_tot", "<u2"),
                            ("q_max_flags", "<u2"), ("sigma_pad_fix", "<u2"), ("sigma_time_fix", "<u2")])
assert DIGIT_DTYPE.itemsize == 8 and CLUSTER_DTYPE.itemsize == 32 and CLUSTER16_DTYPE.itemsize == 16


class tpcclus_params(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("n_sectors", C.c_uint32), ("n_rows", C.c_uint32),
                ("n_time", C.c_uint32), ("n_pads", C.POINTER(C.c_uint16)), ("thr_peak", C.c_uint16),
                ("noise_eps", C.c_uint16), ("max_digits", C.c_uint64), ("flags", C.c_uint32),
                ("device", C.c_int32), ("workspace", C.c_void_p), ("workspace_bytes", C.c_uint64)]


class tpcclus_out(C.Structure):
    _fields_ = [("clusters", C.c_void_p), ("capacity", C.c_uint64), ("n_clusters", C.c_void_p),
                ("status", C.c_void_p)]


class tpcclus_out_packed(C.Structure):
    _fields_ = [("clusters", C.c_void_p), ("capacity", C.c_uint64), ("n_clusters", C.c_void_p),
                ("status", C.c_void_p), ("row_index", C.c_void_p)]


class TpcclusError(RuntimeError):
    def __init__(self, code, what, detail=""):
        super().__init__("%s: %s (%d)%s" % (what, lib().tpcclus_error_string(code).decode(), code,
                                            (": " + detail) if detail else ""))
        self.code = code


_lib = None

EXPORTS = ("tpcclus_workspace_bytes", "tpcclus_workspace_bytes_host", "tpcclus_create", "tpcclus_run",
           "tpcclus_run_host", "tpcclus_destroy", "tpcclus_error_string", "tpcclus_last_error",
           "tpcclus_launches_per_run", "tpcclus_set_timing", "tpcclus_last_timing", "tpcclus_rtc_build_ms",
           "tpcclus_debug_dense_map", "tpcclus_debug_det_fallback", "tpcclus_set_rtc_cache_dir", "tpcclus_rtc_cache_hit", "tpcclus_run_packed",
           "tpcclus_update_params", "tpcclus_constant_buffers", "tpcclus_loaded_units", "tpcclus_debug_shrink",
           "tpcclus_workspace_bytes_host_pipelined", "tpcclus_host_submit", "tpcclus_host_wait", "tpcclus_pack_noalloc")
NOALLOC_MAX_ROWS = 65536   # include/tpcclus.h: TPCCLUS_NOALLOC_MAX_ROWS


def lib() -> C.CDLL:
    """Loads the in-tree library; fails loudly if it has not been built (no fallback)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise ImportError("libtpcclus.so is not built: run `python -m paper_2511_17018_b200.build` "
                          "(or __graft_entry__.build()); there is no CPU fallback")
    L = C.CDLL(_LIB_PATH)
    P = C.POINTER
    L.tpcclus_workspace_bytes.restype = C.c_uint64
    L.tpcclus_workspace_bytes.argtypes = [P(tpcclus_params)]
    L.tpcclus_workspace_bytes_host.restype = C.c_uint64
    L.tpcclus_workspace_bytes_host.argtypes = [P(tpcclus_params), C.c_uint64]
    L.tpcclus_create.restype = C.c_int
    L.tpcclus_create.argtypes = [P(tpcclus_params), P(C.c_void_p)]
    L.tpcclus_run.restype = C.c_int
    L.tpcclus_run.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64, P(tpcclus_out), C.c_int, C.c_void_p]
    L.tpcclus_run_packed.restype = C.c_int
    L.tpcclus_run_packed.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64, P(tpcclus_out_packed), C.c_void_p]
    L.tpcclus_pack_noalloc.restype = C.c_int
    L.tpcclus_pack_noalloc.argtypes = [C.c_void_p, C.c_uint64, C.c_uint32, C.c_uint32, C.c_void_p, C.c_void_p, C.c_void_p,
                                       C.c_char_p, C.c_uint32]
    L.tpcclus_run_host.restype = C.c_int
    L.tpcclus_run_host.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64, C.c_void_p, C.c_uint64,
                                   P(C.c_uint64), P(C.c_uint32), C.c_int, C.c_void_p]
    L.tpcclus_destroy.restype = C.c_int
    L.tpcclus_destroy.argtypes = [C.c_void_p]
    L.tpcclus_error_string.restype = C.c_char_p
    L.tpcclus_error_string.argtypes = [C.c_int]
    L.tpcclus_last_error.restype = C.c_char_p
    L.tpcclus_last_error.argtypes = [C.c_void_p]
    L.tpcclus_launches_per_run.restype = C.c_int
    L.tpcclus_launches_per_run.argtypes = [C.c_void_p, C.c_int]
    L.tpcclus_set_timing.restype = C.c_int
    L.tpcclus_set_timing.argtypes = [C.c_void_p, C.c_int]
    L.tpcclus_last_timing.restype = C.c_int
    L.tpcclus_last_timing.argtypes = [C.c_void_p, P(C.c_char_p), P(C.c_float), C.c_int]
    L.tpcclus_rtc_build_ms.restype = C.c_double
    L.tpcclus_rtc_build_ms.argtypes = [C.c_void_p]
    L.tpcclus_debug_dense_map.restype = C.c_int
    L.tpcclus_debug_dense_map.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
    L.tpcclus_set_rtc_cache_dir.restype = C.c_int
    L.tpcclus_set_rtc_cache_dir.argtypes = [C.c_char_p]
    L.tpcclus_rtc_cache_hit.restype = C.c_int
    L.tpcclus_rtc_cache_hit.argtypes = [C.c_void_p]
    L.tpcclus_debug_det_fallback.restype = C.c_int
    L.tpcclus_debug_det_fallback.argtypes = [C.c_void_p]
    L.tpcclus_workspace_bytes_host_pipelined.restype = C.c_uint64
    L.tpcclus_workspace_bytes_host_pipelined.argtypes = [P(tpcclus_params), C.c_uint64]
    L.tpcclus_host_submit.restype = C.c_int
    L.tpcclus_host_submit.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64, C.c_void_p, C.c_uint64, C.c_int]
    L.tpcclus_host_wait.restype = C.c_int
    L.tpcclus_host_wait.argtypes = [C.c_void_p, P(C.c_uint64), P(C.c_uint32)]
    L.tpcclus_update_params.restype = C.c_int
    L.tpcclus_update_params.argtypes = [C.c_void_p, C.c_uint16, C.c_uint16, C.c_void_p]
    L.tpcclus_constant_buffers.restype = C.c_int
    L.tpcclus_constant_buffers.argtypes = [C.c_void_p]
    L.tpcclus_loaded_units.restype = C.c_int
    L.tpcclus_loaded_units.argtypes = [C.c_void_p, P(C.c_char_p), C.c_int]
    L.tpcclus_debug_shrink.restype = C.c_int
    L.tpcclus_debug_shrink.argtypes = [C.c_void_p, C.c_uint32, C.c_uint64]
    _lib = L
    return L


def make_params(n_sectors, n_rows, n_time, n_pads, max_digits, thr_peak=6, noise_eps=4, flags=0, device=0,
                workspace=0, workspace_bytes=0):
    """Returns (params, keepalive): the n_pads array must outlive the struct."""
    pads = (C.c_uint16 * int(n_rows))(*[int(x) for x in n_pads])
    p = tpcclus_params(C.sizeof(tpcclus_params), int(n_sectors), int(n_rows), int(n_time),
                       C.cast(pads, C.POINTER(C.c_uint16)), int(thr_peak), int(noise_eps), int(max_digits),
                       int(flags), int(device), C.c_void_p(workspace), int(workspace_bytes))
    return p, pads


# ---- same-name wrappers ----------------------------------------------------------------------
def tpcclus_workspace_bytes(params) -> int:
    return int(lib().tpcclus_workspace_bytes(C.byref(params)))


def tpcclus_workspace_bytes_host(params, cluster_capacity) -> int:
    return int(lib().tpcclus_workspace_bytes_host(C.byref(params), int(cluster_capacity)))


def tpcclus_create(params) -> C.c_void_p:
    h = C.c_void_p()
    rc = lib().tpcclus_create(C.byref(params), C.byref(h))
    if rc != 0:
        raise TpcclusError(rc, "tpcclus_create", (lib().tpcclus_last_error(None) or b"").decode())
    return h


def tpcclus_run(handle, d_digits_ptr, n, out: tpcclus_out, mode, stream_ptr) -> None:
    rc = lib().tpcclus_run(handle, C.c_void_p(d_digits_ptr), int(n), C.byref(out), int(mode), C.c_void_p(stream_ptr))
    if rc != 0:
        raise TpcclusError(rc, "tpcclus_run", (lib().tpcclus_last_error(handle) or b"").decode())


def tpcclus_set_rtc_cache_dir(path) -> None:
    lib().tpcclus_set_rtc_cache_dir(None if path is None else os.fsencode(path))


def tpcclus_destroy(handle) -> None:
    lib().tpcclus_destroy(handle)


def tpcclus_pack_noalloc(clusters_ptr: int, n: int, n_sectors: int, n_rows: int, packed_ptr: int, row_index_ptr: int,
                         stream: int = 0) -> None:
    """include/tpcclus.h: tpcclus_pack_noalloc -- the packed 16-byte records and the per-row index of an ordered
    cluster list on the device, without a handle, a workspace or any allocation (DEVICE pointers as integers)."""
    err = C.create_string_buffer(256)
    rc = lib().tpcclus_pack_noalloc(C.c_void_p(clusters_ptr), n, n_sectors, n_rows, C.c_void_p(packed_ptr),
                                    C.c_void_p(row_index_ptr), C.c_void_p(stream), err, 256)
    if rc != 0:
        raise TpcclusError(rc, "tpcclus_pack_noalloc", err.value.decode())


class Clusterizer:
    """One handle + the torch tensors that own its device memory."""

    def __init__(self, n_sectors, n_rows, n_time, n_pads, max_digits, thr_peak=6, noise_eps=4, rtc=False,
                 device=0, host_capacity=0, cog_gated=False, cog_shared=False, host_pipelined=False):
        import torch

        if not torch.cuda.is_available():
            raise RuntimeError("tpcclus needs a CUDA device (sm_100a); there is no CPU fallback")
        self._torch = torch
        self.device = torch.device("cuda", device)
        self.n_sectors, self.n_rows, self.n_time = int(n_sectors), int(n_rows), int(n_time)
        self.n_pads = np.asarray(n_pads, dtype=np.uint16).copy()
        self.max_digits = int(max(1, max_digits))
        self.host_capacity = int(host_capacity)
        flags = (RTC if rtc else 0) | (COG_GATED if cog_gated else 0) | (COG_SHARED if cog_shared else 0)
        p, self._pads_keep = make_params(n_sectors, n_rows, n_time, self.n_pads, self.max_digits, thr_peak, noise_eps,
                                         flags, device)
        if host_capacity and host_pipelined:
            nbytes = int(lib().tpcclus_workspace_bytes_host_pipelined(C.byref(p), int(host_capacity)))
        else:
            nbytes = tpcclus_workspace_bytes_host(p, host_capacity) if host_capacity else tpcclus_workspace_bytes(p)
        if nbytes == 0:
            raise TpcclusError(-1, "tpcclus_workspace_bytes", "invalid or unsupported parameters")
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        p.workspace = self.workspace.data_ptr()
        p.workspace_bytes = nbytes
        self.workspace_bytes = nbytes
        self._params = p
        self._h = tpcclus_create(p)
        self._n = torch.zeros(1, dtype=torch.int64, device=self.device)
        self._status = torch.zeros(1, dtype=torch.int32, device=self.device)

    # -- device path -------------------------------------------------------------------------
    def run(self, digits, mode=MODE_FAST, clusters=None, capacity=None, stream=None):
        """digits: int64/uint8 CUDA tensor of packed 8-byte records.  Enqueues and returns
        (clusters uint8[cap,32], n_clusters int64[1], status int32[1]) without synchronising."""
        torch = self._torch
        n = digits.numel() if digits.dtype == torch.int64 else digits.numel() // 8
        assert digits.is_cuda and digits.is_contiguous()
        if clusters is None:
            cap = int(capacity if capacity is not None else max(n, 1))
            clusters = torch.empty((cap, 32), dtype=torch.uint8, device=self.device)
        cap = clusters.shape[0]
        out = tpcclus_out(clusters.data_ptr(), cap, self._n.data_ptr(), self._status.data_ptr())
        st = (stream or torch.cuda.current_stream(self.device)).cuda_stream
        tpcclus_run(self._h, digits.data_ptr(), n, out, mode, st)
        return clusters, self._n, self._status

    def run_sync(self, digits, mode=MODE_FAST, capacity=None):
        """run() + synchronise + copy back: (numpy clusters[CLUSTER_DTYPE], n_clusters, status)."""
        cl, n, st = self.run(digits, mode, capacity=capacity)
        self._torch.cuda.synchronize(self.device)
        n_true, status = int(n.item()), int(st.item())
        m = min(n_true, cl.shape[0])
        return cl[:m].cpu().numpy().view(CLUSTER_DTYPE).reshape(-1), n_true, status

    def run_packed(self, digits, clusters=None, capacity=None, stream=None):
        """Deterministic path, packed output: (clusters uint8[cap,16], row_index int64[S*R+1],
        n_clusters int64[1], status int32[1]); enqueues without synchronising."""
        torch = self._torch
        n = digits.numel() if digits.dtype == torch.int64 else digits.numel() // 8
        assert digits.is_cuda and digits.is_contiguous()
        if clusters is None:
            cap = int(capacity if capacity is not None else max(n, 1))
            clusters = torch.empty((cap, 16), dtype=torch.uint8, device=self.device)
        ridx = torch.empty(self.n_sectors * self.n_rows + 1, dtype=torch.int64, device=self.device)
        out = tpcclus_out_packed(clusters.data_ptr(), clusters.shape[0], self._n.data_ptr(), self._status.data_ptr(),
                                 ridx.data_ptr())
        st = (stream or torch.cuda.current_stream(self.device)).cuda_stream
        rc = lib().tpcclus_run_packed(self._h, C.c_void_p(digits.data_ptr()), n, C.byref(out), C.c_void_p(st))
        if rc != 0:
            raise TpcclusError(rc, "tpcclus_run_packed", (lib().tpcclus_last_error(self._h) or b"").decode())
        return clusters, ridx, self._n, self._status

    # -- host path (e2e) -----------------------------------------------------------------------
    def run_host(self, digits_host, clusters_host, mode=MODE_FAST, stream=None):
        """digits_host / clusters_host: host tensors or numpy arrays (pinned preferred).
        Synchronous.  Returns (n_clusters, status); clusters_host[:min(n,cap)] is filled."""
        torch = self._torch
        dptr, n = _host_ptr_count(digits_host, 8)
        cptr, cap = _host_ptr_count(clusters_host, 32)
        assert cap <= self.host_capacity, "create the Clusterizer with host_capacity >= len(clusters_host)"
        n_out, status = C.c_uint64(0), C.c_uint32(0)
        st = (stream or torch.cuda.current_stream(self.device)).cuda_stream
        rc = lib().tpcclus_run_host(self._h, C.c_void_p(dptr), n, C.c_void_p(cptr), cap, C.byref(n_out),
                                    C.byref(status), int(mode), C.c_void_p(st))
        if rc != 0:
            raise TpcclusError(rc, "tpcclus_run_host", (lib().tpcclus_last_error(self._h) or b"").decode())
        return int(n_out.value), int(status.value)

    def host_submit(self, digits_host, clusters_host, mode=MODE_FAST):
        """tpcclus_host_submit: one more frame into the two-deep host pipeline (host_pipelined=True handles)."""
        dptr, n = _host_ptr_count(digits_host, 8)
        cptr, cap = _host_ptr_count(clusters_host, 32)
        rc = lib().tpcclus_host_submit(self._h, C.c_void_p(dptr), n, C.c_void_p(cptr), cap, int(mode))
        if rc != 0:
            raise TpcclusError(rc, "tpcclus_host_submit", (lib().tpcclus_last_error(self._h) or b"").decode())

    def host_wait(self):
        """tpcclus_host_wait: (n_clusters, status) of the oldest frame in flight; its clusters are in the buffer given at submit."""
        n_out, status = C.c_uint64(0), C.c_uint32(0)
        rc = lib().tpcclus_host_wait(self._h, C.byref(n_out), C.byref(status))
        if rc != 0:
            raise TpcclusError(rc, "tpcclus_host_wait", (lib().tpcclus_last_error(self._h) or b"").decode())
        return int(n_out.value), int(status.value)

    # -- introspection ---------------------------------------------------------------------------
    def launches_per_run(self, mode):
        return int(lib().tpcclus_launches_per_run(self._h, int(mode)))

    def set_timing(self, enable=True):
        lib().tpcclus_set_timing(self._h, 1 if enable else 0)

    def last_timing(self):
        names = (C.c_char_p * 16)()
        ms = (C.c_float * 16)()
        k = lib().tpcclus_last_timing(self._h, names, ms, 16)
        if k < 0:
            raise TpcclusError(k, "tpcclus_last_timing")
        return [(names[i].decode(), float(ms[i])) for i in range(k)]

    @property
    def rtc_build_ms(self):
        return float(lib().tpcclus_rtc_build_ms(self._h))

    @property
    def rtc_cache_hit(self):
        return int(lib().tpcclus_rtc_cache_hit(self._h)) == 1

    def update_params(self, thr_peak, noise_eps, stream=None):
        """tpcclus_update_params: new thresholds into every registered constant block, stream-ordered."""
        st = (stream or self._torch.cuda.current_stream(self.device)).cuda_stream
        rc = lib().tpcclus_update_params(self._h, int(thr_peak), int(noise_eps), C.c_void_p(st))
        if rc != 0:
            raise TpcclusError(rc, "tpcclus_update_params", (lib().tpcclus_last_error(self._h) or b"").decode())

    @property
    def constant_buffers(self):
        return int(lib().tpcclus_constant_buffers(self._h))

    def loaded_units(self):
        names = (C.c_char_p * 32)()
        k = lib().tpcclus_loaded_units(self._h, names, 32)
        return [names[i].decode() for i in range(k)]

    def debug_shrink(self, slice_cap=0, blob_cap=0):
        rc = lib().tpcclus_debug_shrink(self._h, int(slice_cap), int(blob_cap))
        if rc != 0:
            raise TpcclusError(rc, "tpcclus_debug_shrink")

    def dense_map(self, stream=None):
        """Debug hook (step a1): the O0 map of the last run as a flat uint16 CUDA tensor in
        [sector][row][time][pad] order."""
        torch = self._torch
        cells = self.n_sectors * self.n_time * int(self.n_pads.astype(np.int64).sum())
        m = torch.empty(cells, dtype=torch.int16, device=self.device)
        st = (stream or torch.cuda.current_stream(self.device)).cuda_stream
        rc = lib().tpcclus_debug_dense_map(self._h, C.c_void_p(m.data_ptr()), C.c_void_p(st))
        if rc != 0:
            raise TpcclusError(rc, "tpcclus_debug_dense_map", (lib().tpcclus_last_error(self._h) or b"").decode())
        return m

    def det_fallback(self):
        """Debug hook: did the last DETERMINISTIC run take the chained-scan fallback?"""
        return int(lib().tpcclus_debug_det_fallback(self._h)) == 1

    def close(self):
        if getattr(self, "_h", None):
            self._torch.cuda.synchronize(self.device)
            tpcclus_destroy(self._h)
            self._h = None
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def _host_ptr_count(x, itemsize):
    if isinstance(x, np.ndarray):
        assert x.flags["C_CONTIGUOUS"]
        return x.ctypes.data, x.nbytes // itemsize
    assert (not x.is_cuda) and x.is_contiguous()
    return x.data_ptr(), (x.numel() * x.element_size()) // itemsize
