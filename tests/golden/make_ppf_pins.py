"""Recomputes the library-side numbers stored in ppf_pins.json with numpy / scipy only.

    python tests/golden/make_ppf_pins.py            # prints stored vs recomputed, exits 1 on a mismatch

The stored values were first produced by probes of the survey (pins P1-P4) and are cited
there; this script is the committed way to regenerate them.  It imports neither oracle/ nor the CUDA package: the
prototype is scipy.signal.firwin, the filter bank is numpy.fft applied to the folded (polyphase) form, the synthesis
is numpy.convolve per residue -- library routines, not the code under test.  The two PAPER.md quotes in the file
(8 * N_S FLOP per sample, 200e6 complex samples per second) are the paper's own numbers and are not
recomputed."""
from __future__ import annotations

import json
import os
import sys

import numpy as np
from scipy.signal import firwin

M, P = 1024, 16
HERE = os.path.dirname(os.path.abspath(__file__))


def analysis(x, h):
    """Critically sampled PPF, fold + FFT form: Y_m[k] = FFT_M( sum_t h[r + tM] x[(m + t)M + r] )[k]."""
    T = x.size // M - (P - 1)
    hp = h.reshape(P, M)
    xs = x[:(T + P - 1) * M].reshape(T + P - 1, M)
    u = np.zeros((T, M))
    for t in range(P):
        u += hp[t][None, :] * xs[t:t + T]
    return np.fft.fft(u, axis=1)[:, :M // 2]


def synthesis(Y, h):
    """Unnormalised Hermitian inverse DFT (bin 512 zero, Re of bin 0) and the matched FIR g = M h per residue."""
    T = Y.shape[0]
    full = np.zeros((T, M // 2 + 1), dtype=complex)
    full[:, :M // 2] = Y
    y = M * np.fft.irfft(full, M, axis=1)
    g = M * h.reshape(P, M)
    ylead = np.vstack([np.zeros((P - 1, M)), y])
    out = np.zeros((T, M))
    for r in range(M):
        out[:, r] = np.convolve(ylead[:, r], g[:, r])[P - 1:P - 1 + T]
    return out.reshape(-1)


def main() -> int:
    stored = json.load(open(os.path.join(HERE, "ppf_pins.json")))
    h = firwin(P * M, 1.0 / M, window=("kaiser", 9.0))
    hp = h.reshape(P, M)
    dc = M * hp.sum(axis=0)
    en = (M * hp) ** 2
    got = {"P3_max_h": h.max(), "P3_dc_min": dc.min(), "P3_dc_max": dc.max(), "P3_energy_r0": en.sum(axis=0)[0],
           "P3_energy_r511": en.sum(axis=0)[511], "P3_energy_mean": en.sum(axis=0).mean()}
    rng = np.random.default_rng(20161206)
    T = 96
    x = rng.standard_normal((T + P - 1) * M)
    xh = synthesis(analysis(x, h), h)
    ref = x[:T * M]                                   # zero net delay: xhat[n] ~ x[n]
    lo = P * M
    got["P1_rel_l2"] = np.linalg.norm(xh[lo:] - ref[lo:]) / np.linalg.norm(ref[lo:])
    got["P1_gain"] = float(xh[lo:] @ ref[lo:] / (ref[lo:] @ ref[lo:]))
    n = np.arange((T + P - 1) * M)
    for name, k in (("centre", 300.0), ("edge", 300.5)):
        tone = np.cos(2 * np.pi * k * n / M)
        th = synthesis(analysis(tone, h), h)
        if name == "centre":
            got["P2_tone_centre_err"] = np.linalg.norm(th[lo:] - tone[lo:T * M]) / np.linalg.norm(tone[lo:T * M])
        else:
            got["P2_tone_edge_amp"] = np.sqrt(2 * np.mean(th[lo:] ** 2))
    imp = np.zeros((T + P - 1) * M)
    n0 = 40 * M + 377
    imp[n0] = 1.0
    ih = synthesis(analysis(imp, h), h)
    got["P4_impulse_r377"] = {"main": ih[n0], "echo1": ih[n0 + M], "echo2": ih[n0 + 2 * M], "echo3": ih[n0 + 3 * M]}

    bad = 0
    for key, val in got.items():
        s = stored[key]
        if isinstance(val, dict):
            for sub, v in val.items():
                ok = abs(v - s[sub]) <= s["tol"]
                bad += not ok
                print(f"{key}.{sub:6s} stored {s[sub]:+.6f}  recomputed {v:+.6f}  {'ok' if ok else 'MISMATCH'}")
            continue
        if "value" in s:
            ok = abs(val - s["value"]) <= s["tol"]
            print(f"{key:20s} stored {s['value']:.10g} +- {s['tol']:g}  recomputed {val:.10g}  {'ok' if ok else 'MISMATCH'}")
        else:
            ok = s.get("lo", -np.inf) <= val <= s.get("hi", np.inf)
            print(f"{key:20s} stored [{s.get('lo', '-inf')}, {s.get('hi', 'inf')}]  recomputed {val:.6g}  {'ok' if ok else 'MISMATCH'}")
        bad += not ok
    return 1 if bad else 0


if __name__ == "__main__":
    sys.exit(main())
