"""ctypes binding of include/bsh.h -- argument marshalling only."""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np

from . import build as _build

BSH_UNWEIGHTED, BSH_WEIGHTED, BSH_NAIVE = 0, 1, 16
BSH_OPT_KERNEL_FAMILY, BSH_OPT_FORCE_CLAMP, BSH_OPT_PIXELS_PER_THREAD = 1, 2, 3
BSH_FAMILY_AUTO, BSH_FAMILY_PIXEL_LANE, BSH_FAMILY_TEMPLATE_LANE, BSH_FAMILY_WINDOW = 0, 1, 2, 3

EXPORTS = ["bsh_version", "bsh_create", "bsh_destroy", "bsh_last_error", "bsh_get_stats", "bsh_set_option",
           "bsh_measure_peaks", "bsh_build_peakgram", "bsh_normalise_peakgram", "bsh_median_bias",
           "bsh_stage1_hough", "bsh_stage1_launch", "bsh_stage1_collect", "bsh_stage2_power", "bsh_search_patch_host",
           "bsh_template_index", "bsh_template_decode", "bsh_template_index_ecc", "bsh_template_decode_ecc", "bsh_post_coincidences", "bsh_post_cluster",
           "bsh_post_coincidences_static"]

# numpy view of bsh_cand (24 bytes)
CAND_DTYPE = np.dtype([("index", "<u8"), ("count", "<i4"), ("wcount", "<f4"), ("power", "<f4"), ("flags", "<u4")])


class BshError(RuntimeError):
    pass


class _Sfts(C.Structure):
    _fields_ = [("n_sft", C.c_int32), ("t_sft", C.c_double), ("h_t_mid", C.c_void_p), ("h_v_over_c", C.c_void_p),
                ("d_w", C.c_void_p), ("k_slab0", C.c_int64), ("n_bins", C.c_int32), ("t_search_mid", C.c_double)]


class _Grid(C.Structure):
    _fields_ = [("n_pix", C.c_int32), ("h_alpha", C.c_void_p), ("h_delta", C.c_void_p), ("k_band0", C.c_int64),
                ("n_f0", C.c_int32), ("n_ap", C.c_int32), ("h_ap", C.c_void_p), ("n_P", C.c_int32), ("h_P", C.c_void_p),
                ("n_tasc", C.c_int32), ("h_tasc_frac", C.c_void_p),
                ("n_ecc", C.c_int32), ("h_ecosw", C.c_void_p), ("h_esinw", C.c_void_p)]


class _CandSet(C.Structure):
    _fields_ = [("n", C.c_int32), ("d_param", C.c_void_p), ("d_res", C.c_void_p), ("d_sig", C.c_void_p)]


class Stats(C.Structure):
    _fields_ = [("peakgram_ms", C.c_float), ("stage1_setup_ms", C.c_float), ("stage1_kernel_ms", C.c_float),
                ("stage1_select_ms", C.c_float), ("stage2_ms", C.c_float), ("n_templates", C.c_int64),
                ("n_accumulations", C.c_int64), ("n_candidates", C.c_int64), ("threshold", C.c_double),
                ("n_passes", C.c_int32), ("kernel_variant", C.c_int32), ("threads_per_block", C.c_int32),
                ("grid_blocks", C.c_int32), ("launches", C.c_int64), ("host_tables_ms", C.c_float), ("frontend_ms", C.c_float)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


class Peaks(C.Structure):
    _fields_ = [("n_sm", C.c_int32), ("sm_clock_mhz", C.c_double), ("issue_warp_inst_per_clk_smsp", C.c_double),
                ("lop3_lanes_per_clk_sm", C.c_double), ("fadd_lanes_per_clk_sm", C.c_double),
                ("dadd_lanes_per_clk_sm", C.c_double), ("dmul_lanes_per_clk_sm", C.c_double),
                ("lds32_bytes_per_clk_sm", C.c_double), ("lds64_bytes_per_clk_sm", C.c_double),
                ("lds128_bytes_per_clk_sm", C.c_double)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


_lib = None


def library():
    """Load (building if needed) the in-tree libbsh.so.  Raises if it cannot be built or loaded."""
    global _lib
    if _lib is None:
        path = _build.build_library()
        lib = C.CDLL(path)
        lib.bsh_last_error.restype = C.c_char_p
        lib.bsh_template_index.restype = C.c_uint64
        lib.bsh_template_decode.restype = None
        lib.bsh_template_index_ecc.restype = C.c_uint64
        lib.bsh_template_decode_ecc.restype = None
        lib.bsh_median_bias.restype = C.c_double
        for name in EXPORTS:
            getattr(lib, name)                       # fail loudly on a missing symbol
        _lib = lib
    return _lib


class _Problem:
    """Host arrays (kept alive) + the two C structs describing one workload."""

    def __init__(self, wl, d_w=None):
        f64 = lambda a: np.ascontiguousarray(a, np.float64)
        self.a = dict(t_mid=f64(wl.t_mid), v=f64(wl.v_over_c), alpha=f64(wl.alpha), delta=f64(wl.delta), ap=f64(wl.ap),
                      P=f64(wl.P), tf=f64(wl.tasc_frac))
        ecw = getattr(wl, "ecosw", None)
        n_ecc = 0 if ecw is None else len(ecw)
        if n_ecc:
            self.a.update(ecw=f64(ecw), esw=f64(wl.esinw))
        a = self.a
        self.sfts = _Sfts(n_sft=a["t_mid"].shape[0], t_sft=float(wl.t_sft), h_t_mid=a["t_mid"].ctypes.data,
                          h_v_over_c=a["v"].ctypes.data, d_w=(d_w.data_ptr() if d_w is not None else None),
                          k_slab0=int(wl.k_slab0), n_bins=int(wl.n_bins), t_search_mid=float(wl.t_search_mid))
        self.grid = _Grid(n_pix=a["alpha"].shape[0], h_alpha=a["alpha"].ctypes.data, h_delta=a["delta"].ctypes.data,
                          k_band0=int(wl.k_band0), n_f0=int(wl.n_f0), n_ap=a["ap"].shape[0], h_ap=a["ap"].ctypes.data,
                          n_P=a["P"].shape[0], h_P=a["P"].ctypes.data, n_tasc=a["tf"].shape[0],
                          h_tasc_frac=a["tf"].ctypes.data, n_ecc=n_ecc, h_ecosw=a["ecw"].ctypes.data if n_ecc else None,
                          h_esinw=a["esw"].ctypes.data if n_ecc else None)
        self.d_w = d_w


def median_bias(window: int = 101) -> float:
    return float(library().bsh_median_bias(C.c_int32(window)))


def template_index(wl, pix, ia, ip, it, j) -> int:
    return int(library().bsh_template_index(C.byref(_Problem(wl).grid), pix, ia, ip, it, j))


def template_index_ecc(wl, pix, ia, ip, it, ie, j) -> int:
    return int(library().bsh_template_index_ecc(C.byref(_Problem(wl).grid), pix, ia, ip, it, ie, j))


def template_decode_ecc(wl, index):
    out = [C.c_int32() for _ in range(6)]
    library().bsh_template_decode_ecc(C.byref(_Problem(wl).grid), C.c_uint64(int(index)), *[C.byref(o) for o in out])
    return tuple(o.value for o in out)


def template_decode(wl, index):
    out = [C.c_int32() for _ in range(5)]
    library().bsh_template_decode(C.byref(_Problem(wl).grid), C.c_uint64(int(index)), *[C.byref(o) for o in out])
    return tuple(o.value for o in out)


STATIC_MAX_CANDS = 8192        # BSH_STATIC_MAX_CANDS of include/bsh.h


def post_coincidences_static(a, b, window: float, out, device: int = 0, stream=None):
    """bsh_post_coincidences_static: the coincidence step (Eq. 44) for callers that cannot allocate device memory
    -- the GPU's memory belongs to somebody else's pool, other patches' kernels are running and must not be stalled by a
    cudaMalloc, or the answer is needed in bounded time (include/bsh.h gives the full account).  No Context is involved and
    the library allocates nothing: its work area is a fixed array inside the loaded library, which limits each list to
    STATIC_MAX_CANDS = 8192 candidates (BshError with code -6 beyond that) and means that two such calls must never run on
    one GPU at the same time.  This wrapper allocates nothing either.

    a, b: (d_param [n, 6], d_res [n, 6], d_sig [n]) CUDA float64 tensors on `device`.
    out:  the caller's result buffers (pair_a int32 [cap], pair_b int32 [cap], centroid float64 [cap, 6], significance
          float64 [cap]) on `device`; at most cap pairs are written.
    stream: a torch.cuda.Stream, or None for the legacy default stream.
    Returns the number of pairs found (it may exceed cap).  The first call on a device also looks up the work area's address;
    make it at set-up time, before any stream capture."""
    import torch
    lib = library()
    pa, pb, cen, sig = out
    cap = int(pa.shape[0])
    assert pa.is_cuda and pa.dtype == torch.int32 and pb.dtype == torch.int32 and int(pb.shape[0]) == cap
    assert cen.dtype == torch.float64 and tuple(cen.shape) == (cap, 6) and sig.dtype == torch.float64 and int(sig.shape[0]) == cap
    assert all(t.is_contiguous() and t.is_cuda for t in out)
    sets = []
    for d_param, d_res, d_sig in (a, b):
        n = int(d_param.shape[0])
        for t, shape in ((d_param, (n, 6)), (d_res, (n, 6)), (d_sig, (n,))):
            assert t.is_cuda and t.dtype == torch.float64 and tuple(t.shape) == shape and t.is_contiguous()
        sets.append(_CandSet(n=n, d_param=d_param.data_ptr() if n else None, d_res=d_res.data_ptr() if n else None,
                             d_sig=d_sig.data_ptr() if n else None))
    n_pairs = C.c_int64(0)
    err = C.create_string_buffer(512)
    rc = lib.bsh_post_coincidences_static(C.c_int(device), C.c_void_p(stream.cuda_stream if stream is not None else None),
                                          C.byref(sets[0]), C.byref(sets[1]), C.c_double(window), C.c_int64(cap),
                                          C.c_void_p(pa.data_ptr()), C.c_void_p(pb.data_ptr()), C.c_void_p(cen.data_ptr()),
                                          C.c_void_p(sig.data_ptr()), C.byref(n_pairs), err, C.c_int32(len(err)))
    if rc != 0:
        raise BshError(f"bsh error {rc}: {err.value.decode()}")
    return int(n_pairs.value)


class Context:
    """One bsh_ctx bound to a torch CUDA device and stream."""

    def __init__(self, device: int = 0, stream=None):
        import torch
        if not torch.cuda.is_available():
            raise BshError("no CUDA device: the BinarySkyHough path has no CPU fallback")
        self.torch = torch
        self.lib = library()
        self.device = device
        torch.cuda.set_device(device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(device)
        self._ctx = C.c_void_p()
        rc = self.lib.bsh_create(C.byref(self._ctx), C.c_int(device), C.c_void_p(self.stream.cuda_stream))
        if rc != 0:
            raise BshError(f"bsh_create failed ({rc})")
        self._keep = []

    def close(self):
        if self._ctx:
            self.lib.bsh_destroy(self._ctx)
            self._ctx = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc):
        if rc != 0:
            raise BshError(f"bsh error {rc}: {self.lib.bsh_last_error(self._ctx).decode()}")

    def _empty(self, shape, dtype):
        """An output buffer for the library: on the context's device (not torch's current one) and allocated under the
        context's stream, the stream the kernels write it on, so that the caching allocator's reuse rules follow that stream."""
        torch = self.torch
        with torch.cuda.stream(self.stream):
            return torch.empty(shape, dtype=dtype, device=f"cuda:{self.device}")

    # ---- the three calls of the path -------------------------------------------------------------------------------
    def build_peakgram(self, d_rho, rho_th: float = 1.6, out=None):
        """d_rho: CUDA float32 [N, K] (row stride = d_rho.stride(0)).  Returns CUDA int32 tensor [N, ceil(K/32)] holding
        the uint32 bit words."""
        torch = self.torch
        assert d_rho.is_cuda and d_rho.dtype == torch.float32 and d_rho.dim() == 2 and d_rho.stride(1) == 1
        n, k = d_rho.shape
        wpr = (k + 31) // 32
        if out is None:
            out = self._empty((n, wpr), torch.int32)
        self._check(self.lib.bsh_build_peakgram(self._ctx, C.c_void_p(d_rho.data_ptr()), C.c_int32(n), C.c_int32(k),
                                                C.c_int64(d_rho.stride(0)), C.c_float(rho_th), C.c_void_p(out.data_ptr()),
                                                C.c_int32(out.shape[1])))
        return out

    def normalise_peakgram(self, d_sft, window: int = 101, bias=None, rho_th: float = 1.6, want_rho=True, want_peak=True):
        """d_sft: CUDA complex64 [N, n_raw] (row stride = d_sft.stride(0)).  Returns (d_rho float32 [N, K] or None,
        d_peak int32 [N, ceil(K / 32)] or None), K = n_raw - window + 1 (front end, Eq. 20-21 + L176)."""
        torch = self.torch
        assert d_sft.is_cuda and d_sft.dtype == torch.complex64 and d_sft.dim() == 2 and d_sft.stride(1) == 1
        n, n_raw = d_sft.shape
        k = n_raw - window + 1
        b = median_bias(window) if bias is None else bias
        d_rho = self._empty((n, k), torch.float32) if want_rho else None
        d_peak = self._empty((n, (k + 31) // 32), torch.int32) if want_peak else None
        self._check(self.lib.bsh_normalise_peakgram(
            self._ctx, C.c_void_p(d_sft.data_ptr()), C.c_int32(n), C.c_int32(n_raw), C.c_int64(d_sft.stride(0)),
            C.c_int32(window), C.c_float(b), C.c_float(rho_th), C.c_void_p(d_rho.data_ptr() if want_rho else None),
            C.c_int64(k), C.c_void_p(d_peak.data_ptr() if want_peak else None),
            C.c_int32(d_peak.shape[1] if want_peak else 0)))
        return d_rho, d_peak

    def stage1_launch(self, d_peak, wl, mode=BSH_UNWEIGHTED, topk=None, d_w=None, counts_full=None):
        pb = _Problem(wl, d_w)
        topk = int(topk if topk is not None else wl.topk)
        self._pending = (pb, topk)
        self._check(self.lib.bsh_stage1_launch(self._ctx, C.c_void_p(d_peak.data_ptr()), C.c_int32(d_peak.shape[1]),
                                               C.byref(pb.sfts), C.byref(pb.grid), C.c_int32(mode), C.c_int32(topk),
                                               C.c_void_p(counts_full.data_ptr() if counts_full is not None else None)))

    def stage1_collect(self):
        torch = self.torch
        pb, topk = self._pending
        d_top = self._empty(topk * CAND_DTYPE.itemsize, torch.uint8)
        n_top = C.c_int32(0)
        self._check(self.lib.bsh_stage1_collect(self._ctx, C.c_void_p(d_top.data_ptr()), C.byref(n_top)))
        return d_top, int(n_top.value)

    def stage1_hough(self, d_peak, wl, mode=BSH_UNWEIGHTED, topk=None, d_w=None, counts_full=None):
        """Returns (d_top, n_top): d_top is a CUDA uint8 tensor holding topk bsh_cand records (best first)."""
        torch = self.torch
        pb = _Problem(wl, d_w)
        topk = int(topk if topk is not None else wl.topk)
        d_top = self._empty(topk * CAND_DTYPE.itemsize, torch.uint8)
        n_top = C.c_int32(0)
        self._check(self.lib.bsh_stage1_hough(self._ctx, C.c_void_p(d_peak.data_ptr()), C.c_int32(d_peak.shape[1]),
                                              C.byref(pb.sfts), C.byref(pb.grid), C.c_int32(mode), C.c_int32(topk),
                                              C.c_void_p(d_top.data_ptr()), C.byref(n_top),
                                              C.c_void_p(counts_full.data_ptr() if counts_full is not None else None)))
        return d_top, int(n_top.value)

    def stage2_power(self, d_rho, wl, d_cands, n_cands: int, d_w=None, sort_by_power: bool = True):
        pb = _Problem(wl, d_w)
        self._check(self.lib.bsh_stage2_power(self._ctx, C.c_void_p(d_rho.data_ptr()), C.c_int64(d_rho.stride(0)),
                                              C.byref(pb.sfts), C.byref(pb.grid), C.c_void_p(d_cands.data_ptr()),
                                              C.c_int32(n_cands), C.c_int32(int(sort_by_power))))
        return d_cands

    def search_patch_host(self, rho: np.ndarray, w: Optional[np.ndarray], wl, mode=BSH_UNWEIGHTED, topk=None,
                          rho_th: float = 1.6, out: Optional[np.ndarray] = None):
        """End-to-end call on HOST buffers (numpy, ideally pinned): returns (records[topk], n_top)."""
        topk = int(topk if topk is not None else wl.topk)
        pb = _Problem(wl, None)
        if out is None:
            out = np.zeros(topk, CAND_DTYPE)
        n_top = C.c_int32(0)
        wp = None if w is None else C.c_void_p(w.ctypes.data)
        self._check(self.lib.bsh_search_patch_host(self._ctx, C.c_void_p(rho.ctypes.data), wp, C.c_float(rho_th),
                                                   C.byref(pb.sfts), C.byref(pb.grid), C.c_int32(mode), C.c_int32(topk),
                                                   C.c_void_p(out.ctypes.data), C.byref(n_top)))
        return out, int(n_top.value)

    # ---- post-processing of the toplists (section V.E) -------------------------------------------------------------
    def _candset(self, d_param, d_res, d_sig):
        torch = self.torch
        n = int(d_param.shape[0])
        for t, shape in ((d_param, (n, 6)), (d_res, (n, 6)), (d_sig, (n,))):
            assert t.is_cuda and t.dtype == torch.float64 and tuple(t.shape) == shape and t.is_contiguous()
        return _CandSet(n=n, d_param=d_param.data_ptr() if n else None, d_res=d_res.data_ptr() if n else None,
                        d_sig=d_sig.data_ptr() if n else None)

    def post_coincidences(self, a, b, window: float, max_pairs=None):
        """a, b: (d_param [n, 6], d_res [n, 6], d_sig [n]) CUDA float64 tensors.  Returns (pair_a, pair_b, centroid [m, 6],
        significance [m]) CUDA tensors, pairs in (a, b) order (Eq. 44)."""
        torch = self.torch
        ca, cb = self._candset(*a), self._candset(*b)
        cap = int(max_pairs if max_pairs is not None else max(1, min(ca.n * cb.n, 1 << 22)))
        while True:
            pa, pb = self._empty(cap, torch.int32), self._empty(cap, torch.int32)
            cen, sig = self._empty((cap, 6), torch.float64), self._empty(cap, torch.float64)
            n = C.c_int64(0)
            self._check(self.lib.bsh_post_coincidences(self._ctx, C.byref(ca), C.byref(cb), C.c_double(window), C.c_int64(cap),
                                                       C.c_void_p(pa.data_ptr()), C.c_void_p(pb.data_ptr()),
                                                       C.c_void_p(cen.data_ptr()), C.c_void_p(sig.data_ptr()), C.byref(n)))
            if n.value <= cap or max_pairs is not None:
                m = min(n.value, cap)
                return pa[:m], pb[:m], cen[:m], sig[:m]
            cap = int(n.value)

    def post_cluster(self, cands, window: float, prune_window: float = 0.0):
        """cands: (d_param, d_res, d_sig).  Returns dict(label [n], root, centroid [c, 6], significance, n_members, best)."""
        torch = self.torch
        c = self._candset(*cands)
        n = max(c.n, 1)
        label, root, members = (self._empty(n, torch.int32) for _ in range(3))
        cen, sig = self._empty((n, 6), torch.float64), self._empty(n, torch.float64)
        nc, best = C.c_int32(0), C.c_int32(-1)
        self._check(self.lib.bsh_post_cluster(self._ctx, C.byref(c), C.c_double(window), C.c_double(prune_window),
                                              C.c_void_p(label.data_ptr()), C.c_void_p(root.data_ptr()),
                                              C.c_void_p(cen.data_ptr()), C.c_void_p(sig.data_ptr()),
                                              C.c_void_p(members.data_ptr()), C.byref(nc), C.byref(best)))
        k = nc.value
        return dict(label=label[:c.n], root=root[:k], centroid=cen[:k], significance=sig[:k], n_members=members[:k],
                    best=int(best.value))

    def set_option(self, option: int, value: int):
        """Diagnostic switches (kernel family, table geometry); see include/bsh.h."""
        self._check(self.lib.bsh_set_option(self._ctx, C.c_int32(option), C.c_int32(value)))

    def measure_peaks(self) -> dict:
        """Measured on-chip peak rates of this device (bsh_measure_peaks)."""
        pk = Peaks()
        self._check(self.lib.bsh_measure_peaks(self._ctx, C.byref(pk)))
        return pk.as_dict()

    def stats(self) -> dict:
        s = Stats()
        self._check(self.lib.bsh_get_stats(self._ctx, C.byref(s)))
        return s.as_dict()

    @staticmethod
    def records(d_top, n=None) -> np.ndarray:
        """CUDA uint8 record buffer -> numpy structured array."""
        a = d_top.cpu().numpy().view(CAND_DTYPE)
        return a if n is None else a[:n]
