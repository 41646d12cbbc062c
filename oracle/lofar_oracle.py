"""ctypes binding of the CPU oracle (oracle/lofar_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this module.  It imports nothing from paper_1612_06592_b200 and the CUDA
library imports nothing from here.

The C file holds the arithmetic (definitions O0..O8, each citing the passage of
PAPER.md / BASELINE.json it follows).  This module only marshals numpy arrays and
strings the steps together in the paper's order:
beamform (+ de-dispersion phase) -> inverse DFT -> synthesis FIR -> envelope -> candidates.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lofar_oracle.c")
_LIB = os.path.join(_HERE, "liblofar_oracle.so")

CI8, CI16 = 0, 1


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (portable -O2, OpenMP; never tuned)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(
            ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-fvisibility=hidden",
             "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        c = ctypes
        vp, i, ll, d = c.c_void_p, c.c_int, c.c_longlong, c.c_double
        _lib.lofar_oracle_threads.restype = i
        _lib.lofar_oracle_prototype.argtypes = [i, i, d, vp]
        _lib.lofar_oracle_ppf_analysis.argtypes = [vp, i, i, vp, i, vp]
        _lib.lofar_oracle_tables.argtypes = [i, i, i, i, i, i, d, d, vp, vp, vp, vp]
        _lib.lofar_oracle_beamform.argtypes = [vp, i, i, i, ll, i, i, vp, vp, ll, ll, vp]
        _lib.lofar_oracle_idft.argtypes = [vp, i, i, i, ll, vp]
        _lib.lofar_oracle_synthesis.argtypes = [vp, i, i, vp, ll, vp]
        _lib.lofar_oracle_envelope.argtypes = [vp, ll, i, vp]
        _lib.lofar_oracle_envelope.restype = d
        _lib.lofar_oracle_candidates.argtypes = [vp, vp, i, ll, d, ll, vp, vp]
        _lib.lofar_oracle_candidates.restype = ll
    return _lib


def _p(a: np.ndarray) -> int:
    assert a.flags["C_CONTIGUOUS"]
    return a.ctypes.data


def threads() -> int:
    return int(lib().lofar_oracle_threads())


# --------------------------------------------------------------------------- steps
def prototype(M: int = 1024, P: int = 16, beta: float = 9.0) -> np.ndarray:
    """O0: Kaiser-windowed sinc prototype h[M*P], sum(h) = 1."""
    h = np.empty(M * P, dtype=np.float64)
    lib().lofar_oracle_prototype(M, P, float(beta), _p(h))
    return h


def ppf_analysis(x: np.ndarray, h: np.ndarray, M: int, P: int, T: int) -> np.ndarray:
    """O1 (direct form): real x[(T+P-1)*M] -> Y[T][M/2] complex."""
    x = np.ascontiguousarray(x, dtype=np.float64)
    assert x.size >= (T + P - 1) * M and h.size == M * P
    Y = np.empty((T, M // 2), dtype=np.complex128)
    lib().lofar_oracle_ppf_analysis(_p(x), M, P, _p(np.ascontiguousarray(h)), T, _p(Y))
    return Y


def tables(tau: np.ndarray, stec: np.ndarray, K: int, k0: int, M: int = 1024,
           clock_hz: float = 200e6, f_zone_hz: float = 100e6):
    """O3: W[B][S][K], Dph[D][K]."""
    tau = np.ascontiguousarray(tau, dtype=np.float64)
    stec = np.ascontiguousarray(np.atleast_1d(stec), dtype=np.float64)
    B, S = tau.shape
    D = stec.size
    W = np.empty((B, S, K), dtype=np.complex128)
    Dph = np.empty((D, K), dtype=np.complex128)
    lib().lofar_oracle_tables(S, B, D, K, k0, M, float(clock_hz), float(f_zone_hz),
                              _p(tau), _p(stec), _p(W), _p(Dph))
    return W, Dph


def _dtype_code(X: np.ndarray) -> int:
    if X.dtype == np.int8:
        return CI8
    if X.dtype == np.int16:
        return CI16
    raise TypeError("X must be int8 or int16")


def beamform(X: np.ndarray, W: np.ndarray, Dph: np.ndarray, q0: int = 0, nq: int | None = None):
    """O4: X[S][2][K][T][2] ints -> Z[B*D][K][nq] complex128 for slices q0..q0+nq-1."""
    S, two, K, T, c = X.shape
    assert two == 2 and c == 2
    B = W.shape[0]
    D = Dph.shape[0]
    assert W.shape == (B, S, K) and Dph.shape == (D, K)
    nq = T - q0 if nq is None else nq
    assert 0 <= q0 and q0 + nq <= T
    Z = np.empty((B * D, K, nq), dtype=np.complex128)
    lib().lofar_oracle_beamform(_p(X), _dtype_code(X), S, K, T, B, D,
                                _p(np.ascontiguousarray(W)), _p(np.ascontiguousarray(Dph)),
                                q0, nq, _p(Z))
    return Z


def idft(Z1: np.ndarray, k0: int, M: int = 1024) -> np.ndarray:
    """O5: one series Z1[K][nq] -> y[nq][M] (naive Hermitian inverse DFT, unnormalised)."""
    Z1 = np.ascontiguousarray(Z1, dtype=np.complex128)
    K, nq = Z1.shape
    assert k0 >= 0 and k0 + K <= M // 2
    y = np.empty((nq, M), dtype=np.float64)
    lib().lofar_oracle_idft(_p(Z1), K, k0, M, nq, _p(y))
    return y


def synthesis(ylead: np.ndarray, h: np.ndarray, M: int = 1024, P: int = 16) -> np.ndarray:
    """O6: ylead[(P-1)+nq][M] (P-1 history slices first) -> xhat[nq*M]."""
    ylead = np.ascontiguousarray(ylead, dtype=np.float64)
    nq = ylead.shape[0] - (P - 1)
    assert nq >= 0 and ylead.shape[1] == M
    out = np.empty(nq * M, dtype=np.float64)
    lib().lofar_oracle_synthesis(_p(ylead), M, P, _p(np.ascontiguousarray(h)), nq, _p(out))
    return out


def envelope(x: np.ndarray, Wn: int = 1, lead: np.ndarray | None = None):
    """O7: returns (env[N], sigma).  lead = the Wn-1 samples before the block (zeros if None)."""
    x = np.asarray(x, dtype=np.float64)
    if lead is None:
        lead = np.zeros(Wn - 1)
    assert lead.size == Wn - 1
    xl = np.ascontiguousarray(np.concatenate([np.asarray(lead, dtype=np.float64), x]))
    env = np.empty(x.size, dtype=np.float64)
    sigma = lib().lofar_oracle_envelope(_p(xl), x.size, Wn, _p(env))
    return env, float(sigma)


def candidates(env: np.ndarray, sigma: np.ndarray, kappa: float, cap: int = 1 << 22):
    """O8 for one beam: env[D][N], sigma[D] -> (samples[int64], trials[int32], true count)."""
    env = np.ascontiguousarray(np.atleast_2d(env), dtype=np.float64)
    sigma = np.ascontiguousarray(np.atleast_1d(sigma), dtype=np.float64)
    D, N = env.shape
    sample = np.empty(cap, dtype=np.int64)
    trial = np.empty(cap, dtype=np.int32)
    n = lib().lofar_oracle_candidates(_p(env), _p(sigma), D, N, float(kappa), cap,
                                      _p(sample), _p(trial))
    m = min(n, cap)
    return sample[:m].copy(), trial[:m].copy(), int(n)


# --------------------------------------------------------------------------- the chain
@dataclass
class Candidate:
    series: int
    trial: int
    sample: int   # global 5 ns index = stream_offset + q*M + r
    env: float
    sigma: float


@dataclass
class OraclePipeline:
    """The whole hot path, step by step, with the streaming state of reading A12:
    the last P-1 inverse-DFT slices per series and the last Wn-1 output samples per series."""
    tau: np.ndarray            # [B][S] seconds
    stec: np.ndarray           # [D] TECU
    K: int
    k0: int
    M: int = 1024
    P: int = 16
    beta: float = 9.0
    clock_hz: float = 200e6
    f_zone_hz: float = 100e6
    kappa: float = 6.0
    Wn: int = 1
    h: np.ndarray | None = None
    W: np.ndarray = field(init=False)
    Dph: np.ndarray = field(init=False)

    def __post_init__(self):
        self.tau = np.atleast_2d(np.asarray(self.tau, dtype=np.float64))
        self.stec = np.atleast_1d(np.asarray(self.stec, dtype=np.float64))
        self.B, self.S = self.tau.shape
        self.D = self.stec.size
        if self.h is None:
            self.h = prototype(self.M, self.P, self.beta)
        self.W, self.Dph = tables(self.tau, self.stec, self.K, self.k0, self.M,
                                  self.clock_hz, self.f_zone_hz)
        self.reset()

    @property
    def nseries(self) -> int:
        return self.B * self.D

    def reset(self):
        self.yhist = np.zeros((self.nseries, self.P - 1, self.M))
        self.xtail = np.zeros((self.nseries, max(self.Wn - 1, 0)))
        self.offset = 0

    # -- windows (used for sampled parity at full size) -------------------------------
    def yhat(self, X: np.ndarray, series: int, q0: int, nq: int) -> np.ndarray:
        """O4 + O5 for one series and slices q0..q0+nq-1 of block X."""
        b, d = divmod(series, self.D)
        Z = beamform(X, self.W[b:b + 1], self.Dph[d:d + 1], q0, nq)
        return idft(Z[0], self.k0, self.M)

    def series_window(self, X: np.ndarray, series: int, q0: int, nq: int,
                      yhist: np.ndarray | None = None) -> np.ndarray:
        """xhat for slices q0..q0+nq-1 of one series of block X.  Slices before the block come
        from yhist[P-1][M] (the carried history; zeros if None)."""
        Pm = self.P - 1
        lo = max(q0 - Pm, 0)
        y = self.yhat(X, series, lo, q0 + nq - lo)
        need = Pm - (q0 - lo)
        if need > 0:
            hist = np.zeros((Pm, self.M)) if yhist is None else yhist
            y = np.concatenate([hist[Pm - need:], y], axis=0)
        return synthesis(y, self.h, self.M, self.P)

    # -- one whole block, streaming state carried ---------------------------------------
    def run_block(self, X: np.ndarray, want_series: bool = True):
        """Returns (series[nseries][T*M] or None, sigma[nseries], list[Candidate], true count)."""
        T = X.shape[3]
        N = T * self.M
        Z = beamform(X, self.W, self.Dph)
        series = np.empty((self.nseries, N))
        envs = np.empty((self.nseries, N))
        sigma = np.empty(self.nseries)
        for n in range(self.nseries):
            y = idft(Z[n], self.k0, self.M)
            ylead = np.concatenate([self.yhist[n], y], axis=0)
            series[n] = synthesis(ylead, self.h, self.M, self.P)
            self.yhist[n] = ylead[ylead.shape[0] - (self.P - 1):]
            envs[n], sigma[n] = envelope(series[n], self.Wn, self.xtail[n])
            if self.Wn > 1:
                self.xtail[n] = np.concatenate([self.xtail[n], series[n]])[-(self.Wn - 1):]
        cands: list[Candidate] = []
        total = 0
        for b in range(self.B):
            sl = slice(b * self.D, (b + 1) * self.D)
            smp, trl, cnt = candidates(envs[sl], sigma[sl], self.kappa)
            total += cnt
            for n_, d_ in zip(smp.tolist(), trl.tolist()):
                sidx = b * self.D + d_
                cands.append(Candidate(sidx, d_, self.offset + n_, float(envs[sidx, n_]),
                                       float(sigma[sidx])))
        self.offset += N
        return (series if want_series else None), sigma, cands, total
