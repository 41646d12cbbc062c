"""ctypes binding of the CPU oracle (oracle/lofar_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this module.  It imports nothing from paper_1612_06592_b200 and the CUDA
library imports nothing from here.

The C file holds the arithmetic of the north_star path (definitions O0..O10, each citing the
passage of PAPER.md / BASELINE.json it follows).  This module marshals numpy arrays, strings the
steps together in the paper's order:
beamform (+ de-dispersion phase) -> inverse DFT -> synthesis FIR -> envelope -> candidates,
and holds, in plain numpy (fp64), the definitions of the rows "next" of SURVEY.md 8(f):
O11 LSMR inversion of the polyphase filter (f1), O12 exact paper-order de-dispersion (f2),
O13 re-quantisation between the two beamforming stages (f4).
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
    """Compile the oracle with gcc (portable -O2, OpenMP; never tuned).

    LOFAR_ORACLE_SANITIZE=1 builds and loads an AddressSanitizer + UBSan copy instead (run the pins as
    `LD_PRELOAD=$(gcc -print-file-name=libasan.so) ASAN_OPTIONS=detect_leaks=0 LOFAR_ORACLE_SANITIZE=1 python -m pytest
    tests/test_oracle_pins.py tests/test_oracle_next_pins.py`)."""
    san = os.environ.get("LOFAR_ORACLE_SANITIZE") == "1"
    out = _LIB.replace(".so", "_san.so") if san else _LIB
    flags = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer"] \
        if san else ["-O2"]
    if force or not os.path.exists(out) or os.path.getmtime(out) < os.path.getmtime(_SRC):
        tmp = out + f".tmp{os.getpid()}"
        subprocess.check_call(
            ["gcc", *flags, "-std=c11", "-fopenmp", "-fPIC", "-shared", "-fvisibility=hidden",
             "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, out)
    return out


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


def set_threads(n: int):
    lib().lofar_oracle_set_threads(int(n))


BUILD_FLAGS = "gcc -O2 -std=c11 -fopenmp (portable: the built library travels between machines)"


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
    the last P-1 inverse-DFT slices per series and the last Wn-1 output samples per series.

    Options for the rows "next" (defaults = the north_star path):
      inversion = "matched" (O6) | "lsmr" (O11, lsmr_iters iterations)
      dedisp    = "subband" (phase per sub-band folded into the beam weight, O3/O4) |
                  "exact"   (O12: beams formed without dispersion phase, the reconstructed 5 ns series
                             de-dispersed per trial; output one slice behind the input)
      sigma_mode = "block" (O7: sigma of this block) | "causal" (O9: sigma of the previous block;
                   block 0 uses sigma_init if given, else its own sigma)"""
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
    inversion: str = "matched"
    lsmr_iters: int = 25
    dedisp: str = "subband"
    sigma_mode: str = "block"
    sigma_init: np.ndarray | None = None
    W: np.ndarray = field(init=False)
    Dph: np.ndarray = field(init=False)

    def __post_init__(self):
        self.tau = np.atleast_2d(np.asarray(self.tau, dtype=np.float64))
        self.stec = np.atleast_1d(np.asarray(self.stec, dtype=np.float64))
        self.B, self.S = self.tau.shape
        self.D = self.stec.size
        if self.h is None:
            self.h = prototype(self.M, self.P, self.beta)
        tab_stec = np.zeros(1) if self.dedisp == "exact" else self.stec
        self.W, self.Dph = tables(self.tau, tab_stec, self.K, self.k0, self.M,
                                  self.clock_hz, self.f_zone_hz)
        self.reset()

    @property
    def nseries(self) -> int:
        return self.B * self.D

    @property
    def ninv(self) -> int:
        """Series that go through the inverse PPF: one per beam in exact mode, else one per (beam, trial)."""
        return self.B if self.dedisp == "exact" else self.nseries

    def reset(self):
        self.yhist = np.zeros((self.ninv, self.P - 1, self.M))
        self.xtail = np.zeros((self.nseries, max(self.Wn - 1, 0)))
        self.xprev2 = np.zeros((self.B, 2 * self.M))        # exact mode: last two slices of xhat per beam
        self.sigma_prev = None
        self.last_sigma_ref = None
        self.offset = 0

    def invert(self, ylead: np.ndarray) -> np.ndarray:
        if self.inversion == "lsmr":
            return lsmr_inversion(ylead, self.h, self.lsmr_iters, self.M, self.P)
        return synthesis(ylead, self.h, self.M, self.P)

    # -- windows (used for sampled parity at full size) -------------------------------
    def yhat(self, X: np.ndarray, series: int, q0: int, nq: int) -> np.ndarray:
        """O4 + O5 for one series and slices q0..q0+nq-1 of block X."""
        b, d = divmod(series, self.D)
        Z = beamform(X, self.W[b:b + 1], self.Dph[d:d + 1], q0, nq)
        return idft(Z[0], self.k0, self.M)

    def series_window(self, X: np.ndarray, series: int, q0: int, nq: int,
                      yhist: np.ndarray | None = None) -> np.ndarray:
        """xhat for slices q0..q0+nq-1 of one series of block X (matched synthesis, sub-band phases).
        Slices before the block come from yhist[P-1][M] (the carried history; zeros if None)."""
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
        for n in range(self.ninv):
            y = idft(Z[n], self.k0, self.M)
            ylead = np.concatenate([self.yhist[n], y], axis=0)
            xhat = self.invert(ylead)
            self.yhist[n] = ylead[ylead.shape[0] - (self.P - 1):]
            if self.dedisp == "exact":
                xl = np.concatenate([self.xprev2[n], xhat])
                for d in range(self.D):
                    series[n * self.D + d] = dedisperse_exact(xl, self.stec[d], self.M, self.clock_hz, self.f_zone_hz)
                self.xprev2[n] = xl[xl.size - 2 * self.M:]
            else:
                series[n] = xhat
        for n in range(self.nseries):
            envs[n], sigma[n] = envelope(series[n], self.Wn, self.xtail[n])
            if self.Wn > 1:
                self.xtail[n] = np.concatenate([self.xtail[n], series[n]])[-(self.Wn - 1):]
        # O9: the level candidates are measured against
        if self.sigma_mode == "causal":
            if self.sigma_prev is not None:
                ref = self.sigma_prev
            elif self.sigma_init is not None:
                ref = np.asarray(self.sigma_init, dtype=np.float64)
            else:
                ref = sigma
        else:
            ref = sigma
        self.sigma_prev = sigma.copy()
        self.last_sigma_ref = np.array(ref, dtype=np.float64)
        cands: list[Candidate] = []
        total = 0
        for b in range(self.B):
            sl = slice(b * self.D, (b + 1) * self.D)
            smp, trl, cnt = candidates(envs[sl], ref[sl], self.kappa)
            total += cnt
            for n_, d_ in zip(smp.tolist(), trl.tolist()):
                sidx = b * self.D + d_
                cands.append(Candidate(sidx, d_, self.offset + n_, float(envs[sidx, n_]),
                                       float(ref[sidx])))
        self.offset += N
        return (series if want_series else None), sigma, cands, total


# =========================================================================== rows "next"
def cluster(beam, sample, snr, gap: int):
    """O10 (f3): events from one block's candidate list (beams one after the other, samples increasing).
    Returns a list of dicts: beam, first, last, count, peak (index into the input list)."""
    beam = np.ascontiguousarray(beam, dtype=np.int32)
    sample = np.ascontiguousarray(sample, dtype=np.int64)
    snr = np.ascontiguousarray(snr, dtype=np.float64)
    n = beam.size
    cap = max(n, 1)
    first = np.empty(cap, dtype=np.int64); last = np.empty(cap, dtype=np.int64)
    count = np.empty(cap, dtype=np.int64); peak = np.empty(cap, dtype=np.int64)
    L = lib()
    L.lofar_oracle_cluster.argtypes = [ctypes.c_void_p] * 3 + [ctypes.c_longlong] * 3 + [ctypes.c_void_p] * 4
    L.lofar_oracle_cluster.restype = ctypes.c_longlong
    nev = L.lofar_oracle_cluster(_p(beam), _p(sample), _p(snr), n, int(gap), cap, _p(first), _p(last), _p(count), _p(peak))
    return [dict(beam=int(beam[peak[i]]), first=int(first[i]), last=int(last[i]), count=int(count[i]),
                 peak=int(peak[i])) for i in range(int(nev))]


def ppf_system(h: np.ndarray, r: int, nq: int, M: int = 1024, P: int = 16) -> np.ndarray:
    """The paper's FIR system H for residue r ("a system of sparse linear equations H x^ = y
    where H is the matrix of the FIR filters"), dense, for pins and brute force.  Rows: the nq slices of
    y (row m <-> y[m][r]/M); columns: nq + P - 1 slices of the unknown series x[(m + t) M + r]:
        y[m][r] / M = sum_{t=0}^{P-1} h[r + t M] * x_r[m + t]            (O1 after the inverse DFT)."""
    A = np.zeros((nq, nq + P - 1))
    for m in range(nq):
        for t in range(P):
            A[m, m + t] = h[r + t * M]
    return A


def lsmr_inversion(ylead: np.ndarray, h: np.ndarray, iters: int = 25, M: int = 1024, P: int = 16) -> np.ndarray:
    """O11 (f1): least-squares inversion of the polyphase filter by LSMR ("This system is
    solved by an iterative LSMR algorithm [14] ... convergence ... after approximately 25 iterations";
    Fong & Saunders), reading A23:
      * H is block diagonal over the M residues, so each residue r is its own system (ppf_system):
        rows = the P-1 carried slices and the nq slices of this block (ylead, as for O6), unknowns =
        slices -(P-1) .. nq+P-2 of x_r; the nq slices 0..nq-1 are the output (zero net delay, as O6);
      * x0 = 0, no damping, exactly `iters` iterations, no stopping test.
    The recurrences are those of the LSMR paper, section "Algorithm LSMR", written for all residues at
    once (every scalar is an array over r; nothing couples the residues).
    ylead: [(P-1)+nq][M] -> xhat[nq*M]."""
    ylead = np.ascontiguousarray(ylead, dtype=np.float64)
    n_eq = ylead.shape[0]
    nq = n_eq - (P - 1)
    n_un = n_eq + P - 1
    taps = np.asarray(h, dtype=np.float64).reshape(P, M)          # taps[t][r] = h[r + t M]

    def A_mul(v):                       # [n_un][M] -> [n_eq][M]:  (A v)[m] = sum_t taps[t] v[m + t]
        out = np.zeros((n_eq, M))
        for t in range(P):
            out += taps[t][None, :] * v[t:t + n_eq]
        return out

    def At_mul(u):                      # [n_eq][M] -> [n_un][M]:  (A^T u)[n] = sum_t taps[t] u[n - t]
        out = np.zeros((n_un, M))
        for t in range(P):
            out[t:t + n_eq] += taps[t][None, :] * u
        return out

    def normalise(w):
        nrm = np.sqrt((w * w).sum(axis=0))
        return nrm, np.divide(w, nrm[None, :], out=np.zeros_like(w), where=nrm[None, :] > 0)

    b = ylead / float(M)
    beta, u = normalise(b)
    alpha, v = normalise(At_mul(u))
    alphabar = alpha.copy()
    zetabar = alpha * beta
    rho = np.ones(M); rhobar = np.ones(M); cbar = np.ones(M); sbar = np.zeros(M)
    hvec = v.copy(); hbar = np.zeros_like(v); x = np.zeros_like(v)
    safe = lambda a, d: np.divide(a, d, out=np.zeros_like(a), where=d != 0)
    for _ in range(iters):
        beta, u = normalise(A_mul(v) - alpha[None, :] * u)
        alpha, v_next = normalise(At_mul(u) - beta[None, :] * v)
        rhoold = rho
        rho = np.hypot(alphabar, beta)
        c = safe(alphabar, rho); s = safe(beta, rho)
        thetanew = s * alpha
        alphabar = c * alpha
        rhobarold = rhobar
        thetabar = sbar * rho
        rhotemp = cbar * rho
        rhobar = np.hypot(rhotemp, thetanew)
        cbar = safe(rhotemp, rhobar); sbar = safe(thetanew, rhobar)
        zeta = cbar * zetabar
        zetabar = -sbar * zetabar
        hbar = hvec - safe(thetabar * rho, rhoold * rhobarold)[None, :] * hbar
        x = x + safe(zeta, rho * rhobar)[None, :] * hbar
        hvec = v_next - safe(thetanew, rho)[None, :] * hvec
        v = v_next
    return np.ascontiguousarray(x[P - 1:P - 1 + nq]).reshape(-1)


SEG_SLICES, SEG_GUARD = 16, 1          # O12: overlap-save segment and guard, in slices


def dedisperse_factor(stec: float, nfft: int, clock_hz: float = 200e6, f_zone_hz: float = 100e6) -> np.ndarray:
    """O12 table: D[j] = exp(-2 pi i * 1.343e9 * STEC / f_j), f_j = f_zone + j * clock / nfft, j = 0..nfft/2,
    for the half spectrum of an nfft-point real transform of the 5 ns series (reading A2: baseband bin j of
    the series is sky frequency f_zone + j clock/nfft).  The two self-conjugate bins 0 and nfft/2 keep
    only the real part of the phasor so that the output stays real."""
    j = np.arange(nfft // 2 + 1)
    f = f_zone_hz + j * (clock_hz / nfft)
    turns = np.mod(1.343e9 * stec / f, 1.0)
    D = np.exp(-2j * np.pi * turns)
    D[0] = D[0].real
    D[-1] = D[-1].real
    return D


def dedisperse_exact(xlead: np.ndarray, stec: float, M: int = 1024, clock_hz: float = 200e6,
                     f_zone_hz: float = 100e6) -> np.ndarray:
    """O12 (f2): exact, paper-order de-dispersion of the reconstructed 5 ns series ("the
    signal is Fourier transformed, multiplied in frequency domain by a complex weight depending on the
    STEC value and then transformed back"), reading A24: overlap-save with segments of SEG_SLICES slices
    of which SEG_GUARD slices at either end are discarded (the de-dispersion chirp of the HBA band is
    shorter than one slice for STEC <= 40 TECU); the FFT is a library primitive (numpy.fft).
    xlead: [(2 + T) * M] = the last two slices of the previous block (zeros at stream start) followed
    by the T slices of this block.  Returns y[T * M]: y slice q = de-dispersed xlead slice q + 1, i.e.
    the output runs one slice (5.12 us) behind the input."""
    xlead = np.asarray(xlead, dtype=np.float64)
    T = xlead.size // M - 2
    nfft = SEG_SLICES * M
    keep = SEG_SLICES - 2 * SEG_GUARD
    D = dedisperse_factor(stec, nfft, clock_hz, f_zone_hz)
    y = np.zeros(T * M)
    for q0 in range(0, T, keep):                         # output slices q0 .. q0+keep-1
        seg = np.zeros(nfft)
        lo = q0 * M                                      # xlead slice q0 is the guard slice of this segment
        hi = min(lo + nfft, xlead.size)
        seg[:hi - lo] = xlead[lo:hi]
        out = np.fft.irfft(np.fft.rfft(seg) * D, nfft)
        n = min(keep, T - q0) * M
        y[q0 * M:q0 * M + n] = out[SEG_GUARD * M:SEG_GUARD * M + n]
    return y


def requantise(Z: np.ndarray, scale: float) -> np.ndarray:
    """O13 (f4, two-stage beamforming): the first-stage beams leave the first cluster as 16-bit
    integers: X2 = clip(rint(Z * scale), -32767, 32767), ties to even.
    Z: complex [...]; returns int16 [..., 2]."""
    v = np.stack([Z.real, Z.imag], axis=-1) * scale
    return np.clip(np.rint(v), -32767, 32767).astype(np.int16)
