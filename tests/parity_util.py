"""Helpers shared by the GPU parity tests: tolerances of BASELINE.json:north_star and the
candidate-set comparison rule.  Imports the oracle (tests may) and the
binding; holds no arithmetic of the method itself."""
from __future__ import annotations

import numpy as np

REL_L2 = 1e-5          # "relative L2 error <= 1e-5"
MAX_ABS_RMS = 1e-4     # "max abs error <= 1e-4 * RMS"
GUARD = 1e-4           # trigger guard band, relative to the threshold


def assert_close(got: np.ndarray, ref: np.ndarray, what: str = ""):
    got = np.asarray(got, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    assert got.shape == ref.shape, (what, got.shape, ref.shape)
    assert np.all(np.isfinite(got)), what
    nrm = np.linalg.norm(ref.ravel())
    rms = nrm / np.sqrt(ref.size) if ref.size else 0.0
    err = np.abs(got - ref)
    rel = np.linalg.norm(err.ravel()) / nrm if nrm > 0 else np.linalg.norm(err.ravel())
    mx = err.max() if err.size else 0.0
    assert rel <= REL_L2, f"{what}: rel-L2 {rel:.3e} > {REL_L2}"
    assert mx <= MAX_ABS_RMS * rms + 1e-30, f"{what}: max-abs {mx:.3e} > 1e-4 * RMS ({rms:.3e})"
    return rel, mx / rms if rms > 0 else 0.0


def oracle_snr(oracle, series: np.ndarray, Wn: int, tails=None):
    """env[nseries][N], sigma[nseries] from the oracle's O7 on an oracle series."""
    ns, N = series.shape
    env = np.empty_like(series)
    sigma = np.empty(ns)
    for s in range(ns):
        lead = None if tails is None else tails[s]
        env[s], sigma[s] = oracle.envelope(series[s], Wn, lead)
    return env, sigma


def check_candidates(rec: np.ndarray, total: int, env: np.ndarray, sigma: np.ndarray, B: int, D: int,
                     kappa: float, offset: int = 0):
    """rec: structured GPU records (all stored); env/sigma: the oracle's.  Sets must agree outside the
    guard band; records must be sorted by (beam, sample) and carry consistent fields."""
    N = env.shape[1]
    snr = env / sigma[:, None]
    snr_b = snr.reshape(B, D, N)
    best = snr_b.max(axis=1)                      # [B][N]
    arg = snr_b.argmax(axis=1)
    definite = best > kappa * (1 + GUARD)
    possible = best > kappa * (1 - GUARD)
    assert total == rec.size, "candidate buffer overflowed in a parity test"
    beams = (rec["series"] // D).astype(np.int64)
    samples = rec["sample"].astype(np.int64) - offset
    assert np.all((samples >= 0) & (samples < N))
    got = np.zeros((B, N), dtype=bool)
    got[beams, samples] = True
    assert got.sum() == rec.size, "duplicate (beam, sample) candidates"
    missing = definite & ~got
    extra = got & ~possible
    assert not missing.any(), f"{missing.sum()} oracle candidates missing on the GPU"
    assert not extra.any(), f"{extra.sum()} GPU candidates the oracle rejects"
    # order
    key = beams * N + samples
    assert np.all(np.diff(key) > 0), "candidates not sorted by (beam, sample)"
    # fields
    assert np.all(rec["trial"] == rec["series"] % D)
    tr = rec["trial"].astype(np.int64)
    for i in range(rec.size):
        b, n, d = beams[i], samples[i], tr[i]
        if d != arg[b, n]:
            top = np.sort(snr_b[b, :, n])[::-1]
            assert abs(top[0] - snr_b[b, d, n]) <= GUARD * top[0], "wrong best trial"
        s = b * D + d
        assert abs(rec["env"][i] - env[s, n]) <= 1e-4 * max(env[s, n], sigma[s])
        assert abs(rec["sigma"][i] - sigma[s]) <= 1e-5 * sigma[s]
    return int(definite.sum()), int(got.sum())
