"""Thin ctypes binding of the C-ABI library (include/lofar_moon.h).  Argument marshalling only:
every step of the path runs in the CUDA kernels behind the boundary.  Same names as the C calls.

torch is used for device memory and streams (tensors in, tensors out); nothing here computes.
`load()` fails loudly if liblofar_moon.so is missing -- there is no CPU fallback.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "liblofar_moon.so")

LOFAR_OK, LOFAR_E_INVALID, LOFAR_E_SHAPE, LOFAR_E_ALIGN, LOFAR_E_ALLOC, LOFAR_E_CUDA, \
    LOFAR_E_OVERFLOW, LOFAR_E_STATE = range(8)
LOFAR_CI8, LOFAR_CI16 = 0, 1
LOFAR_SIGMA_BLOCK, LOFAR_SIGMA_CAUSAL = 0, 1
LOFAR_INV_MATCHED, LOFAR_INV_LSMR = 0, 1
LOFAR_DEDISP_SUBBAND, LOFAR_DEDISP_EXACT = 0, 1

# numpy view of lofar_candidate (24 bytes)
CANDIDATE_DTYPE = np.dtype([("series", "<u4"), ("trial", "<u4"), ("sample", "<u8"),
                            ("env", "<f4"), ("sigma", "<f4")])
assert CANDIDATE_DTYPE.itemsize == 24
# numpy view of lofar_event (48 bytes)
EVENT_DTYPE = np.dtype([("beam", "<u4"), ("count", "<u4"), ("first_sample", "<u8"), ("last_sample", "<u8"),
                        ("peak_sample", "<u8"), ("peak_trial", "<u4"), ("peak_env", "<f4"), ("peak_sigma", "<f4"),
                        ("peak_snr", "<f4")])
assert EVENT_DTYPE.itemsize == 48

EXPORTS = (
    "lofar_plan_create", "lofar_plan_destroy", "lofar_plan_set_band", "lofar_plan_set_delays",
    "lofar_plan_set_trials", "lofar_plan_set_filter", "lofar_plan_set_input",
    "lofar_plan_set_trigger", "lofar_plan_set_sigma_mode", "lofar_plan_set_inversion", "lofar_plan_set_dedispersion",
    "lofar_cluster", "lofar_requantize",
    "lofar_plan_workspace_bytes", "lofar_plan_set_allocator",
    "lofar_plan_set_scratch_limit", "lofar_plan_set_overlap", "lofar_plan_chunking", "lofar_plan_chunk_info",
    "lofar_stream_state_bytes",
    "lofar_stream_get_state", "lofar_stream_set_state", "lofar_beamform_dedisperse",
    "lofar_inverse_ppf", "lofar_trigger", "lofar_run_block", "lofar_stream_reset",
    "lofar_stream_push", "lofar_stream_sync", "lofar_plan_profile", "lofar_plan_profile_read",
    "lofar_plan_launch_count", "lofar_status_string", "lofar_trigger_static",
)


class LofarError(RuntimeError):
    def __init__(self, status: int, call: str):
        self.status = status
        super().__init__(f"{call}: {status_string(status)} (status {status})")


_lib = None


def load() -> ctypes.CDLL:
    """Load liblofar_moon.so (build it with `python -m paper_1612_06592_b200.build`)."""
    global _lib
    if _lib is not None:
        return _lib
    path = os.environ.get("LOFAR_MOON_LIB", LIB_PATH)      # ablation builds of build.py; default: the in-tree library
    if not os.path.exists(path):
        raise RuntimeError(f"{path} is missing: build it with `python -m paper_1612_06592_b200.build` "
                           "(there is no CPU fallback)")
    lib = ctypes.CDLL(path)
    c = ctypes
    vp, i, d, u32, u64 = c.c_void_p, c.c_int, c.c_double, c.c_uint32, c.c_uint64
    sig = {
        "lofar_plan_create": (i, [c.POINTER(vp), i, i, i, i, d]),
        "lofar_plan_destroy": (None, [vp]),
        "lofar_plan_set_band": (i, [vp, i, d, d, i]),
        "lofar_plan_set_delays": (i, [vp, vp]),
        "lofar_plan_set_trials": (i, [vp, i, vp]),
        "lofar_plan_set_filter": (i, [vp, vp]),
        "lofar_plan_set_input": (i, [vp, i, i]),
        "lofar_plan_set_trigger": (i, [vp, d, i, u32]),
        "lofar_plan_set_sigma_mode": (i, [vp, i, vp]),
        "lofar_plan_set_inversion": (i, [vp, i, i]),
        "lofar_plan_set_dedispersion": (i, [vp, i]),
        "lofar_cluster": (i, [vp, vp, vp, u64, vp, vp, u32, vp]),
        "lofar_requantize": (i, [vp, vp, i, c.c_float, vp, vp]),
        "lofar_plan_workspace_bytes": (i, [vp, c.POINTER(c.c_size_t)]),
        "lofar_plan_set_allocator": (i, [vp, vp, vp, vp]),
        "lofar_plan_set_scratch_limit": (i, [vp, c.c_size_t]),
        "lofar_plan_set_overlap": (i, [vp, i, i]),
        "lofar_plan_chunking": (i, [vp, i, c.POINTER(c.c_int64), c.POINTER(i), c.POINTER(i)]),
        "lofar_plan_chunk_info": (i, [vp, i, i, c.POINTER(c.c_int64), c.POINTER(c.c_int64), c.POINTER(i), c.POINTER(i)]),
        "lofar_stream_state_bytes": (i, [vp, c.POINTER(c.c_size_t)]),
        "lofar_stream_get_state": (i, [vp, vp, c.c_size_t]),
        "lofar_stream_set_state": (i, [vp, vp, c.c_size_t]),
        "lofar_beamform_dedisperse": (i, [vp, vp, i, vp, vp]),
        "lofar_inverse_ppf": (i, [vp, vp, i, vp, vp]),
        "lofar_trigger": (i, [vp, vp, i, vp, vp, vp, vp]),
        "lofar_run_block": (i, [vp, vp, i, vp, vp, vp, vp, vp]),
        "lofar_stream_reset": (i, [vp]),
        "lofar_stream_push": (i, [vp, vp, i, vp, vp, vp, vp]),
        "lofar_stream_sync": (i, [vp]),
        "lofar_plan_profile": (i, [vp, i]),
        "lofar_plan_profile_read": (i, [vp, vp, vp]),
        "lofar_plan_launch_count": (u64, [vp]),
        "lofar_status_string": (c.c_char_p, [i]),
        "lofar_trigger_static": (i, [vp, i, c.c_int64, c.c_int64, d, u64, vp, u32, vp, vp, vp]),
    }
    for name, (res, args) in sig.items():
        f = getattr(lib, name)
        f.restype = res
        f.argtypes = args
    _lib = lib
    return lib


def status_string(status: int) -> str:
    return load().lofar_status_string(int(status)).decode()


def _check(status: int, call: str, allow=()):
    if status != LOFAR_OK and status not in allow:
        raise LofarError(status, call)
    return status


def _ptr(t) -> int:
    """Device (or pinned host) address of a torch tensor / numpy array; None -> NULL."""
    if t is None:
        return None
    if isinstance(t, np.ndarray):
        assert t.flags["C_CONTIGUOUS"]
        return t.ctypes.data
    assert t.is_contiguous()
    return t.data_ptr()


def _stream_ptr(stream) -> int:
    if stream is None:
        import torch
        stream = torch.cuda.current_stream()
    return stream.cuda_stream or None


class Plan:
    """Owns one lofar_plan*.  Methods carry the names of the C calls they forward to."""

    def __init__(self, stations: int, subbands: int, beams: int, taps: int = 16, stec_tecu: float = 0.0):
        self._lib = load()
        h = ctypes.c_void_p()
        _check(self._lib.lofar_plan_create(ctypes.byref(h), stations, subbands, beams, taps, float(stec_tecu)),
               "lofar_plan_create")
        self._h = h
        self.S, self.K, self.B, self.D = stations, subbands, beams, 1
        self.max_candidates = 65536

    # -- lifetime
    def destroy(self):
        if getattr(self, "_h", None):
            self._lib.lofar_plan_destroy(self._h)
            self._h = None
            self._alloc_thunks = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    @property
    def nseries(self) -> int:
        return self.B * self.D

    # -- setters
    def set_band(self, first_subband: int, f_zone_hz: float = 100e6, clock_hz: float = 200e6, fft_size: int = 1024):
        _check(self._lib.lofar_plan_set_band(self._h, first_subband, f_zone_hz, clock_hz, fft_size), "lofar_plan_set_band")

    def set_delays(self, tau_s):
        tau = np.ascontiguousarray(tau_s, dtype=np.float64)
        assert tau.shape == (self.B, self.S)
        _check(self._lib.lofar_plan_set_delays(self._h, tau.ctypes.data), "lofar_plan_set_delays")

    def set_trials(self, stec_tecu):
        st = np.ascontiguousarray(np.atleast_1d(stec_tecu), dtype=np.float64)
        _check(self._lib.lofar_plan_set_trials(self._h, st.size, st.ctypes.data), "lofar_plan_set_trials")
        self.D = int(st.size)

    def set_filter(self, h=None):
        if h is None:
            _check(self._lib.lofar_plan_set_filter(self._h, None), "lofar_plan_set_filter")
        else:
            hh = np.ascontiguousarray(h, dtype=np.float64)
            assert hh.size == 16 * 1024
            _check(self._lib.lofar_plan_set_filter(self._h, hh.ctypes.data), "lofar_plan_set_filter")

    def set_input(self, dtype: int, max_slices: int):
        _check(self._lib.lofar_plan_set_input(self._h, dtype, max_slices), "lofar_plan_set_input")

    def set_trigger(self, kappa: float, env_window: int = 1, max_candidates: int = 65536):
        _check(self._lib.lofar_plan_set_trigger(self._h, float(kappa), env_window, max_candidates), "lofar_plan_set_trigger")
        self.max_candidates = max_candidates

    def set_inversion(self, mode: int, iterations: int = 25):
        _check(self._lib.lofar_plan_set_inversion(self._h, mode, iterations), "lofar_plan_set_inversion")

    def set_dedispersion(self, mode: int):
        _check(self._lib.lofar_plan_set_dedispersion(self._h, mode), "lofar_plan_set_dedispersion")

    def set_sigma_mode(self, mode: int, sigma_init=None):
        if sigma_init is None:
            _check(self._lib.lofar_plan_set_sigma_mode(self._h, mode, None), "lofar_plan_set_sigma_mode")
        else:
            si = np.ascontiguousarray(sigma_init, dtype=np.float32)
            assert si.size == self.nseries
            _check(self._lib.lofar_plan_set_sigma_mode(self._h, mode, si.ctypes.data), "lofar_plan_set_sigma_mode")

    def cluster(self, cand, count, gap_samples: int, events, nevents, stream=None):
        """events: device uint8 tensor [max_events][48]; nevents: device int32[1]."""
        _check(self._lib.lofar_cluster(self._h, _ptr(cand), _ptr(count), int(gap_samples), _ptr(events), _ptr(nevents),
                                       events.shape[0], _stream_ptr(stream)), "lofar_cluster")

    def workspace_bytes(self) -> int:
        n = ctypes.c_size_t()
        _check(self._lib.lofar_plan_workspace_bytes(self._h, ctypes.byref(n)), "lofar_plan_workspace_bytes")
        return int(n.value)

    ALLOC_FN = ctypes.CFUNCTYPE(ctypes.c_void_p, ctypes.c_size_t, ctypes.c_void_p)
    FREE_FN = ctypes.CFUNCTYPE(None, ctypes.c_void_p, ctypes.c_void_p)

    def set_allocator(self, alloc=None, free=None):
        """alloc(nbytes) -> device address (0 on failure), free(address); None/None restores cudaMalloc.
        The ctypes thunks are kept alive on the Plan for as long as the library may call them."""
        if alloc is None and free is None:
            _check(self._lib.lofar_plan_set_allocator(self._h, None, None, None), "lofar_plan_set_allocator")
            self._alloc_thunks = None
            return
        a = self.ALLOC_FN(lambda n, ctx: alloc(n) or None)
        f = self.FREE_FN(lambda ptr, ctx: free(ptr))
        _check(self._lib.lofar_plan_set_allocator(self._h, ctypes.cast(a, ctypes.c_void_p),
                                                  ctypes.cast(f, ctypes.c_void_p), None), "lofar_plan_set_allocator")
        self._alloc_thunks = (a, f)

    def set_torch_allocator(self):
        """Plan memory from torch's caching allocator (north_star: "PyTorch used only for device memory")."""
        import torch
        self.set_allocator(torch.cuda.caching_allocator_alloc, torch.cuda.caching_allocator_delete)

    def set_scratch_limit(self, nbytes: int):
        _check(self._lib.lofar_plan_set_scratch_limit(self._h, int(nbytes)), "lofar_plan_set_scratch_limit")

    def set_overlap(self, mode: int, chunk_slices: int = 0):
        _check(self._lib.lofar_plan_set_overlap(self._h, int(mode), int(chunk_slices)), "lofar_plan_set_overlap")

    def chunking(self, slices: int):
        """(slices per scratch chunk, spans per inverse-PPF launch, slices per span)."""
        zc, ns, sl = ctypes.c_int64(), ctypes.c_int(), ctypes.c_int()
        _check(self._lib.lofar_plan_chunking(self._h, slices, ctypes.byref(zc), ctypes.byref(ns), ctypes.byref(sl)),
               "lofar_plan_chunking")
        return int(zc.value), int(ns.value), int(sl.value)

    def chunks(self, slices: int):
        """[(first slice, slices, spans, slices per span)] for every scratch chunk of a block of `slices`."""
        out = []
        while True:
            c0, nc, ns, sl = ctypes.c_int64(), ctypes.c_int64(), ctypes.c_int(), ctypes.c_int()
            _check(self._lib.lofar_plan_chunk_info(self._h, slices, len(out), ctypes.byref(c0), ctypes.byref(nc),
                                                   ctypes.byref(ns), ctypes.byref(sl)), "lofar_plan_chunk_info")
            if nc.value == 0:
                return out
            out.append((int(c0.value), int(nc.value), int(ns.value), int(sl.value)))

    def get_state(self) -> np.ndarray:
        n = ctypes.c_size_t()
        _check(self._lib.lofar_stream_state_bytes(self._h, ctypes.byref(n)), "lofar_stream_state_bytes")
        buf = np.zeros(n.value, dtype=np.uint8)
        _check(self._lib.lofar_stream_get_state(self._h, buf.ctypes.data, buf.size), "lofar_stream_get_state")
        return buf

    def set_state(self, buf: np.ndarray, allow=()):
        buf = np.ascontiguousarray(buf, dtype=np.uint8)
        return _check(self._lib.lofar_stream_set_state(self._h, buf.ctypes.data, buf.size), "lofar_stream_set_state", allow)

    def launch_count(self) -> int:
        return int(self._lib.lofar_plan_launch_count(self._h))

    def profile(self, enable: bool):
        _check(self._lib.lofar_plan_profile(self._h, int(enable)), "lofar_plan_profile")

    def profile_read(self):
        """(ms[5], launches[5]) accumulated since the previous read: beamform, inverse PPF, trigger, LSMR, exact
        de-dispersion."""
        ms = np.zeros(5, dtype=np.float64)
        n = np.zeros(5, dtype=np.uint64)
        _check(self._lib.lofar_plan_profile_read(self._h, ms.ctypes.data, n.ctypes.data), "lofar_plan_profile_read")
        return ms, n

    # -- stage calls (device tensors; raw status codes via `allow` for error-path tests)
    def beamform_dedisperse(self, X, slices: int, Z, stream=None, allow=()):
        return _check(self._lib.lofar_beamform_dedisperse(self._h, _ptr(X), slices, _ptr(Z), _stream_ptr(stream)),
                      "lofar_beamform_dedisperse", allow)

    def requantize(self, Z, slices: int, scale: float, X2, stream=None, allow=()):
        return _check(self._lib.lofar_requantize(self._h, _ptr(Z), slices, float(scale), _ptr(X2), _stream_ptr(stream)),
                      "lofar_requantize", allow)

    def inverse_ppf(self, Z, slices: int, series, stream=None, allow=()):
        return _check(self._lib.lofar_inverse_ppf(self._h, _ptr(Z), slices, _ptr(series), _stream_ptr(stream)),
                      "lofar_inverse_ppf", allow)

    def trigger(self, series, slices: int, cand, count, sigma, stream=None, allow=()):
        return _check(self._lib.lofar_trigger(self._h, _ptr(series), slices, _ptr(cand), _ptr(count), _ptr(sigma),
                                              _stream_ptr(stream)), "lofar_trigger", allow)

    def run_block(self, X, slices: int, series, cand, count, sigma, stream=None, allow=()):
        return _check(self._lib.lofar_run_block(self._h, _ptr(X), slices, _ptr(series), _ptr(cand), _ptr(count),
                                                _ptr(sigma), _stream_ptr(stream)), "lofar_run_block", allow)

    # -- streaming
    def stream_reset(self):
        _check(self._lib.lofar_stream_reset(self._h), "lofar_stream_reset")

    def stream_push(self, X_host, slices: int, series, cand_host=None, count_host=None, sigma_host=None, allow=()):
        return _check(self._lib.lofar_stream_push(self._h, _ptr(X_host), slices, _ptr(series), _ptr(cand_host),
                                                  _ptr(count_host), _ptr(sigma_host)), "lofar_stream_push", allow)

    def stream_sync(self, allow=()):
        return _check(self._lib.lofar_stream_sync(self._h), "lofar_stream_sync", allow)


def plan_for(w, tau) -> Plan:
    """Plan configured for a synth.Workload (marshalling of its parameters, nothing else)."""
    p = Plan(w.S, w.K, w.B, w.P, w.stec[0])
    p.set_band(w.k0)
    p.set_delays(tau)
    if w.D > 1:
        p.set_trials(np.asarray(w.stec, dtype=np.float64))
    p.set_input(LOFAR_CI16 if w.dtype == "ci16" else LOFAR_CI8, w.T)
    p.set_trigger(w.kappa, 1, 65536)
    return p


STATIC_MAX_CHUNKS = 524288       # LOFAR_STATIC_MAX_CHUNKS of include/lofar_moon.h


def trigger_static(series, samples: int, kappa: float, cand, count, sigma, offset: int = 0, stream=None, allow=()):
    """lofar_trigger_static: the allocation-free trigger on series[nseries][pitch] (torch tensors of the caller)."""
    lib = load()
    nseries, pitch = int(series.shape[0]), int(series.stride(0))
    return _check(lib.lofar_trigger_static(_ptr(series), nseries, int(samples), pitch, float(kappa), int(offset), _ptr(cand),
                                           int(cand.shape[0]), _ptr(count), _ptr(sigma), _stream_ptr(stream)),
                  "lofar_trigger_static", allow)


def new_outputs(plan: Plan, slices: int, device="cuda"):
    """Allocate the caller-owned output buffers of run_block as torch tensors."""
    import torch
    series = torch.empty((plan.nseries, slices * 1024), dtype=torch.float32, device=device)
    cand = torch.zeros((plan.max_candidates, 24), dtype=torch.uint8, device=device)
    count = torch.zeros(1, dtype=torch.int32, device=device)
    sigma = torch.zeros(plan.nseries, dtype=torch.float32, device=device)
    return series, cand, count, sigma


def events_to_numpy(events, nevents) -> np.ndarray:
    n = int(nevents.item()) if hasattr(nevents, "item") else int(nevents)
    raw = events.cpu().numpy() if hasattr(events, "cpu") else np.asarray(events)
    rec = raw.reshape(-1).view(EVENT_DTYPE)
    return rec[:min(n, rec.size)].copy()


def candidates_to_numpy(cand, count) -> np.ndarray:
    """Copy the stored candidate records to a structured numpy array (device -> host copy only)."""
    n = int(count.item()) if hasattr(count, "item") else int(count)
    raw = cand.cpu().numpy() if hasattr(cand, "cpu") else np.asarray(cand)
    rec = raw.reshape(-1).view(CANDIDATE_DTYPE)
    return rec[:min(n, rec.size)].copy()
