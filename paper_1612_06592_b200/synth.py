"""Seeded synthetic LOFAR-shaped inputs (the five workloads of BASELINE.json:configs).

This module is the ONLY thing the CUDA path and the CPU oracle have in common: it produces the
integer station data X[S][2][K][T][re,im], the delay table tau[B][S] and the STEC list that both
consume.  It holds none of the method's arithmetic (no beamforming, no inverse PPF, no trigger)
and imports neither the oracle nor the CUDA binding.

What it models is the *upstream* of the hot path (PAPER.md:34
and :82-88): a station polyphase filter bank (analysis), station geometry, a dispersed ns pulse
with per-station geometric delays, and 8/16-bit quantisation.  The analysis filter here is the
station firmware's model (scipy.signal.firwin); tests check it against the oracle's direct form.

Recipe:
  * base seed 1612065920; stream seed = base + 1000*config + 48*block + (2s+p);
    geometry/pulse seed = base + 1000*config + 999.
  * config 0: full time-domain path (noise + pulse -> PPF analysis -> select -> quantise).
  * configs 1-4: iid Gaussian noise drawn directly in the sub-band domain (the distribution the
    configs state) + pulse footprints obtained by analysing a 48-slice time-domain window.
"""
from __future__ import annotations

import math
from concurrent.futures import ThreadPoolExecutor
from dataclasses import dataclass, field, replace

import numpy as np

BASE_SEED = 1612065920
C_LIGHT = 299792458.0
M_FFT = 1024
P_TAPS = 16
CLOCK_HZ = 200e6
F_ZONE_HZ = 100e6
K_DISP = 1.343e9          # phi(f) = 2 pi * K_DISP * STEC / f   (BASELINE.json:configs[0])


@dataclass(frozen=True)
class Workload:
    name: str
    index: int                 # BASELINE.json:configs index (seed offset); 9 for ad-hoc cases
    S: int
    B: int
    K: int
    k0: int
    T: int                     # slices per block
    dtype: str                 # "ci8" | "ci16"
    sigma_in: float
    stec: tuple                # trial list (TECU); D = len
    kappa: float
    n_pulses: int
    pulse_stec: float
    blocks: int = 1
    timedomain: bool = False   # config 0: full time-domain generation
    M: int = M_FFT
    P: int = P_TAPS

    @property
    def D(self) -> int:
        return len(self.stec)

    @property
    def nseries(self) -> int:
        return self.B * self.D

    @property
    def np_dtype(self):
        return np.int8 if self.dtype == "ci8" else np.int16

    @property
    def clip(self) -> int:
        return 127 if self.dtype == "ci8" else 32767

    @property
    def input_bytes(self) -> int:
        return self.S * 2 * self.K * self.T * 2 * np.dtype(self.np_dtype).itemsize

    @property
    def slice_seconds(self) -> float:
        return self.M / CLOCK_HZ


CONFIGS = (
    Workload("tiny", 0, S=4, B=2, K=16, k0=300, T=4096, dtype="ci16", sigma_in=8.0,
             stec=(10.0,), kappa=5.0, n_pulses=1, pulse_stec=10.0, timedomain=True),
    Workload("b1_k244_ci16", 1, S=24, B=1, K=244, k0=256, T=131072, dtype="ci16", sigma_in=16.0,
             stec=(15.0,), kappa=6.0, n_pulses=3, pulse_stec=15.0),
    Workload("b24_k488_ci8", 2, S=24, B=24, K=488, k0=24, T=131072, dtype="ci8", sigma_in=4.0,
             stec=(12.0,), kappa=6.0, n_pulses=5, pulse_stec=12.0),
    Workload("stec_sweep", 3, S=24, B=8, K=488, k0=24, T=65536, dtype="ci8", sigma_in=4.0,
             stec=tuple(float(v) for v in range(5, 21)), kappa=6.0, n_pulses=3, pulse_stec=13.0),
    Workload("streaming", 4, S=24, B=24, K=488, k0=24, T=195312, dtype="ci8", sigma_in=4.0,
             stec=(10.0,), kappa=6.0, n_pulses=20, pulse_stec=10.0, blocks=10),
)


def config(i: int) -> Workload:
    return CONFIGS[i]


def small(name="small", **kw) -> Workload:
    """Ad-hoc small workload for tests (same recipe as configs 1-4)."""
    base = dict(index=9, S=3, B=2, K=12, k0=40, T=64, dtype="ci8", sigma_in=4.0, stec=(10.0,),
                kappa=5.0, n_pulses=1, pulse_stec=10.0)
    base.update(kw)
    return Workload(name, **base)


# ----------------------------------------------------------------------------- geometry
def station_positions(S: int, seed: int) -> np.ndarray:
    """(x, y) uniform in a disc of radius 1 km, z = 0 ("dense core with approximately
    2 km diameter"; reading A17)."""
    rng = np.random.default_rng(seed)
    r = 1000.0 * np.sqrt(rng.random(S))
    a = 2.0 * np.pi * rng.random(S)
    return np.stack([r * np.cos(a), r * np.sin(a), np.zeros(S)], axis=1)


def beam_offsets(B: int, pitch_deg: float = 0.09) -> np.ndarray:
    """Hexagonal lattice, the B points nearest the centre, ties by polar angle (reading A16).
    Returns (dl, dm) in radians, shape [B][2]."""
    pts = []
    for a in range(-6, 7):
        for b in range(-6, 7):
            x = a + 0.5 * b
            y = b * math.sqrt(3.0) / 2.0
            pts.append((round(x * x + y * y, 9), math.atan2(y, x) % (2 * math.pi), x, y))
    pts.sort()
    sel = np.array([[p[2], p[3]] for p in pts[:B]])
    return np.deg2rad(pitch_deg) * sel


def delays(pos: np.ndarray, offsets: np.ndarray, zenith_deg: float = 30.0) -> np.ndarray:
    """Differential geometric delay tau[b][s] = -(r_s . dn_b)/c of a plane wave from the beam's
    direction relative to the pointing centre (readings A3, A4).  Pointing: azimuth 0 (north),
    zenith angle 30 deg; tangent-plane basis e_l = east, e_m = n0 x e_l."""
    z = math.radians(zenith_deg)
    e_l = np.array([1.0, 0.0, 0.0])
    e_m = np.array([0.0, math.cos(z), -math.sin(z)])
    dn = offsets[:, :1] * e_l[None, :] + offsets[:, 1:2] * e_m[None, :]
    return -(dn @ pos.T) / C_LIGHT


def geometry(w: Workload):
    seed = BASE_SEED + 1000 * w.index + 999
    pos = station_positions(w.S, seed)
    off = beam_offsets(w.B)
    return pos, off, delays(pos, off)


# ----------------------------------------------------------------------------- station PPF model
_proto_cache: dict = {}


def station_prototype(M: int = M_FFT, P: int = P_TAPS, beta: float = 9.0) -> np.ndarray:
    """The station filter bank's prototype (input-side model): scipy's Kaiser-windowed sinc."""
    key = (M, P, beta)
    if key not in _proto_cache:
        from scipy.signal import firwin
        _proto_cache[key] = firwin(M * P, 1.0 / M, window=("kaiser", beta))
    return _proto_cache[key]


def station_ppf(x: np.ndarray, T: int, M: int = M_FFT, P: int = P_TAPS, h=None) -> np.ndarray:
    """Critically sampled analysis filter bank of the station (fold + FFT form).
    x: real [(T+P-1)*M] -> Y[T][M/2]."""
    h = station_prototype(M, P) if h is None else h
    hp = h.reshape(P, M)
    xs = x[:(T + P - 1) * M].reshape(T + P - 1, M)
    u = np.zeros((T, M))
    for t in range(P):
        u += hp[t][None, :] * xs[t:t + T]
    return np.fft.fft(u, axis=1)[:, :M // 2]


# ----------------------------------------------------------------------------- pulses
@dataclass(frozen=True)
class Pulse:
    beam: int
    sample: float      # global 5 ns sample index (fractional) on the stream's time axis
    stec: float
    amp: float         # peak of the undispersed band-limited pulse per stream, output units


def pulse_amplitude(w: Workload, snr: float = 12.0) -> float:
    """Per-stream time-domain peak such that the beamformed, reconstructed peak is ~snr sigma
    (reading A18).  Output noise sigma from the closed form P8; chain keeps ~0.85 of the peak."""
    sigma_out = math.sqrt(0.9341 * 4.0 * w.K * 2 * w.S) * w.sigma_in
    return snr * sigma_out / (2 * w.S * 0.85)


def make_pulses(w: Workload) -> list:
    """Seeded pulse list on the global time axis of the stream (all blocks).  For the streaming
    config at least 4 pulses straddle a block boundary and 2 fall in the first 15 slices of a
    block."""
    rng = np.random.default_rng(BASE_SEED + 1000 * w.index + 999 + 1)
    total = w.T * w.blocks
    amp = pulse_amplitude(w)
    out = []
    for i in range(w.n_pulses):
        beam = int(rng.integers(0, w.B))
        if w.blocks > 1 and i < 4:      # footprint (slices q-15..q+1) straddles a block edge
            blk = int(rng.integers(1, w.blocks))
            q = blk * w.T + int(rng.integers(1, 12))
        elif w.blocks > 1 and i < 6:    # inside the first 15 slices of a block
            blk = int(rng.integers(1, w.blocks))
            q = blk * w.T + int(rng.integers(0, 15))
        else:
            q = int(rng.integers(min(64, total // 4), max(total - 64, total // 4 + 1)))
        r = int(rng.integers(0, w.M))
        frac = float(rng.random())
        out.append(Pulse(beam, q * w.M + r + frac, w.pulse_stec, amp))
    return out


def pulse_footprint(w: Workload, pulse: Pulse, tau_s: np.ndarray, nwin: int = 48):
    """Sub-band footprint of one dispersed pulse with per-station delay.
    Builds, per station, the real 5 ns series on a window of nwin slices (band-limited flat
    spectrum over the selected sub-bands, fractional-sample position, delay tau_s and dispersion
    e^{+i phi(f_sky)} applied as phases of the half spectrum), runs the station PPF on it and keeps
    the selected sub-bands.  Returns (first global slice m0, F[S][K][nwin-P+1] complex)."""
    M, P = w.M, w.P
    Nw = nwin * M
    q_p = int(pulse.sample // M)
    m0 = q_p - nwin // 2
    n_local = pulse.sample - m0 * M                    # fractional position inside the window
    j = np.arange(Nw // 2 + 1)
    f_bb = j / Nw                                      # cycles per 5 ns sample
    kf = f_bb * M
    mask = (kf >= w.k0 - 0.5) & (kf < w.k0 + w.K - 0.5)
    f_sky = F_ZONE_HZ + f_bb * CLOCK_HZ
    a0 = pulse.amp * Nw / (2.0 * mask.sum())
    base = a0 * mask * np.exp(-2j * np.pi * f_bb * n_local)
    disp = np.exp(2j * np.pi * ((K_DISP * pulse.stec / f_sky) % 1.0))
    F = np.empty((tau_s.size, w.K, nwin - P + 1), dtype=np.complex128)
    for s, tau in enumerate(tau_s):
        spec = base * disp * np.exp(-2j * np.pi * ((f_sky * tau) % 1.0))
        xw = np.fft.irfft(spec, Nw)
        Y = station_ppf(xw, nwin - P + 1, M, P)
        F[s] = Y[:, w.k0:w.k0 + w.K].T
    return m0, F


# ----------------------------------------------------------------------------- blocks
def _stream_seed(w: Workload, block: int, s: int, p: int) -> int:
    return BASE_SEED + 1000 * w.index + 48 * block + (2 * s + p)


def generate_block(w: Workload, block: int = 0, out: np.ndarray | None = None,
                   threads: int | None = None, tau: np.ndarray | None = None) -> np.ndarray:
    """X[S][2][K][T][2] for one block of a sub-band-domain workload (configs 1-4 and small())."""
    if w.timedomain:
        assert block == 0
        return generate_timedomain(w, tau)
    if tau is None:
        _, _, tau = geometry(w)
    X = np.empty((w.S, 2, w.K, w.T, 2), dtype=w.np_dtype) if out is None else out
    assert X.shape == (w.S, 2, w.K, w.T, 2) and X.dtype == w.np_dtype

    # pulse footprints that touch this block
    prints = []
    nwin = 48
    for pl in make_pulses(w):
        q_p = int(pl.sample // w.M)
        lo, hi = q_p - nwin // 2, q_p - nwin // 2 + (nwin - w.P + 1)
        if hi <= block * w.T or lo >= (block + 1) * w.T:
            continue
        m0, F = pulse_footprint(w, pl, tau[pl.beam], nwin)
        prints.append((m0 - block * w.T, F))

    def fill(sp):
        s, p = divmod(sp, 2)
        rng = np.random.default_rng(_stream_seed(w, block, s, p))
        kstep = max(1, (1 << 22) // max(w.T, 1))
        for ka in range(0, w.K, kstep):
            kb = min(w.K, ka + kstep)
            v = rng.standard_normal((kb - ka, w.T, 2), dtype=np.float32)
            v *= np.float32(w.sigma_in)
            for m0, F in prints:
                a, b = max(m0, 0), min(m0 + F.shape[2], w.T)
                if a < b:
                    seg = F[s, ka:kb, a - m0:b - m0]
                    v[:, a:b, 0] += seg.real.astype(np.float32)
                    v[:, a:b, 1] += seg.imag.astype(np.float32)
            np.rint(v, out=v)
            np.clip(v, -w.clip, w.clip, out=v)
            X[s, p, ka:kb] = v

    n = 2 * w.S
    if threads is None:
        import os
        threads = min(n, os.cpu_count() or 1)
    if threads > 1 and X.nbytes > (1 << 24):
        with ThreadPoolExecutor(threads) as ex:
            list(ex.map(fill, range(n)))
    else:
        for sp in range(n):
            fill(sp)
    return X


def generate_timedomain(w: Workload, tau: np.ndarray | None = None) -> np.ndarray:
    """Config 0: per (s,p) a real 5 ns series of (T+P-1)*M samples = N(0,1) noise + one pulse from
    beam 0's direction, through the station PPF, selected sub-bands scaled to sigma_in and rounded
    (ties to even), clipped."""
    if tau is None:
        _, _, tau = geometry(w)
    M, P, T = w.M, w.P, w.T
    N = (T + P - 1) * M
    pulses = make_pulses(w)
    X = np.empty((w.S, 2, w.K, T, 2), dtype=w.np_dtype)
    h = station_prototype(M, P)
    # per-component std of PPF-filtered unit white noise: sum(h^2)/2 per component
    scale = w.sigma_in / math.sqrt(float(np.sum(h * h)) / 2.0)
    nwin = 48
    for s in range(w.S):
        for p in range(2):
            rng = np.random.default_rng(_stream_seed(w, 0, s, p))
            x = rng.standard_normal(N)
            Y = station_ppf(x, T, M, P)[:, w.k0:w.k0 + w.K].T * scale      # [K][T]
            for pl in pulses:
                m0, F = pulse_footprint(w, pl, tau[pl.beam][s:s + 1], nwin)
                a, b = max(m0, 0), min(m0 + F.shape[2], T)
                Y[:, a:b] += F[0][:, a - m0:b - m0]
            v = np.stack([Y.real, Y.imag], axis=-1)
            X[s, p] = np.clip(np.rint(v), -w.clip, w.clip)
    return X


# ----------------------------------------------------------------------------- stage-level inputs
def random_z(seed: int, nseries: int, K: int, T: int, scale: float = 30.0) -> np.ndarray:
    """Seeded complex64 beam sums Z[nseries][K][T] for testing the inverse PPF on its own
    (white, the level of 48 summed int8 streams)."""
    rng = np.random.default_rng(BASE_SEED + 7000 + seed)
    z = rng.standard_normal((nseries, K, T, 2), dtype=np.float32) * np.float32(scale)
    return z.view(np.complex64).reshape(nseries, K, T)


def random_series(seed: int, nseries: int, N: int, spikes: int = 6, level: float = 9.0) -> np.ndarray:
    """Seeded float32 series[nseries][N]: unit white noise plus a few spikes of +-level (some placed
    at the same sample in several series, some near the block edges) for testing the trigger alone."""
    rng = np.random.default_rng(BASE_SEED + 8000 + seed)
    x = rng.standard_normal((nseries, N), dtype=np.float32)
    for i in range(spikes):
        n = int(rng.integers(0, N)) if i >= 2 else (0 if i == 0 else N - 1)
        amp = level * (1.0 + 0.2 * rng.random())
        for s in range(nseries):
            if i % 2 == 0 or s == int(rng.integers(0, nseries)):
                x[s, n] = np.float32(amp * (1 if rng.random() < 0.5 else -1) * (1.0 + 0.05 * s))
    return x
