"""Pins of the CPU oracle (oracle/lofar_oracle.c) against things other than itself.

Every test here checks an oracle function against a closed form, an invariant, a library special
case (numpy.fft / scipy.signal), brute force written out differently, or a physical property of
the chain -- chosen so that a dropped term, a wrong sign/index or a transposed operand fails at
least one.  Pin ids P1..P10 are those of SURVEY.md section 8(c), restated in DESIGN.md.
No GPU, no CUDA library.
"""
import json
import math
import os

import numpy as np
import pytest

from paper_1612_06592_b200 import synth

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "ppf_pins.json")))
M, P = 1024, 16


@pytest.fixture(scope="module")
def h(oracle):
    return oracle.prototype(M, P, 9.0)


def roundtrip(oracle, x, h_, M_=M, P_=P, k0=0, K=None):
    """O1 (fold+FFT form, checked against the direct form below) -> select -> O5 -> O6."""
    K = M_ // 2 - k0 if K is None else K
    T = x.size // M_ - (P_ - 1)
    Y = synth.station_ppf(x, T, M_, P_, h_)                    # [T][M/2]
    Z = np.ascontiguousarray(Y[:, k0:k0 + K].T)                # [K][T]
    y = oracle.idft(Z, k0, M_)
    ylead = np.concatenate([np.zeros((P_ - 1, M_)), y])
    return oracle.synthesis(ylead, h_, M_, P_)


# ------------------------------------------------------------------ O0 prototype (P3)
def test_prototype_equals_scipy_firwin(oracle, h):
    from scipy.signal import firwin
    ref = firwin(M * P, 1.0 / M, window=("kaiser", 9.0))
    assert np.max(np.abs(h - ref)) < 1e-15
    assert abs(h.sum() - 1.0) < 1e-12
    assert np.max(np.abs(h - h[::-1])) < 1e-16                      # symmetric up to rounding
    assert abs(h.max() - GOLD["P3_max_h"]["value"]) < GOLD["P3_max_h"]["tol"]


def test_prototype_polyphase_sums(h):
    hp = h.reshape(P, M)
    dc = M * hp.sum(0)
    en = M * M * (hp ** 2).sum(0)
    assert abs(dc.min() - GOLD["P3_dc_min"]["value"]) < GOLD["P3_dc_min"]["tol"]
    assert abs(dc.max() - GOLD["P3_dc_max"]["value"]) < GOLD["P3_dc_max"]["tol"]
    assert abs(en[0] - GOLD["P3_energy_r0"]["value"]) < GOLD["P3_energy_r0"]["tol"]
    assert abs(en[511] - GOLD["P3_energy_r511"]["value"]) < GOLD["P3_energy_r511"]["tol"]
    assert abs(en.mean() - GOLD["P3_energy_mean"]["value"]) < GOLD["P3_energy_mean"]["tol"]


def test_prototype_small_sizes_generic(oracle):
    from scipy.signal import firwin
    for m, p, beta in [(8, 2, 5.0), (8, 4, 9.0), (16, 3, 2.5)]:
        ref = firwin(m * p, 1.0 / m, window=("kaiser", beta))
        assert np.max(np.abs(oracle.prototype(m, p, beta) - ref)) < 1e-14


# ------------------------------------------------------------------ O1 analysis
def test_analysis_direct_equals_fold_fft(oracle, h):
    rng = np.random.default_rng(7)
    T = 3
    x = rng.standard_normal((T + P - 1) * M)
    Yd = oracle.ppf_analysis(x, h, M, P, T)
    Yf = synth.station_ppf(x, T, M, P, h)
    assert np.max(np.abs(Yd - Yf)) < 1e-13


def test_analysis_tone_lands_in_its_subband(oracle, h):
    """A complex-exponential pair at the centre of sub-band k gives Y[m][k] = 1/2 (unit DC gain of
    the prototype, no slice-to-slice phase advance because k*M/M is an integer number of cycles)."""
    T, k = 4, 300
    n = np.arange((T + P - 1) * M)
    x = np.cos(2 * np.pi * k * n / M)
    Y = oracle.ppf_analysis(x, h, M, P, T)
    assert np.max(np.abs(Y[:, k] - 0.5)) < 1e-6
    others = np.delete(Y, [k], axis=1)
    assert np.max(np.abs(others)) < 2e-5          # Kaiser beta=9 stop band (about -95 dB)


# ------------------------------------------------------------------ O5 inverse DFT (P6)
def test_idft_equals_numpy_irfft_and_parseval(oracle):
    rng = np.random.default_rng(3)
    nq = 5
    Z = rng.standard_normal((M // 2, nq)) + 1j * rng.standard_normal((M // 2, nq))
    y = oracle.idft(Z, 0, M)
    half = np.concatenate([Z.T, np.zeros((nq, 1))], axis=1)      # bin M/2 = 0 (reading A10)
    ref = M * np.fft.irfft(half, M, axis=1)                      # irfft ignores Im of bin 0
    assert np.max(np.abs(y - ref)) < 1e-10
    pars = M * (Z[0].real ** 2 + 2 * np.sum(np.abs(Z[1:]) ** 2, axis=0))
    assert np.allclose((y ** 2).sum(1), pars, rtol=1e-12)


def test_idft_selected_band_zero_fills(oracle):
    rng = np.random.default_rng(4)
    k0, K, nq = 300, 16, 3
    Z = rng.standard_normal((K, nq)) + 1j * rng.standard_normal((K, nq))
    half = np.zeros((nq, M // 2 + 1), dtype=complex)
    half[:, k0:k0 + K] = Z.T
    assert np.max(np.abs(oracle.idft(Z, k0, M) - M * np.fft.irfft(half, M, axis=1))) < 1e-10


def test_idft_single_bin_is_a_cosine(oracle):
    """Sign of the exponent: Z = e^{i a} in bin k gives 2 cos(2 pi k r / M + a) (inverse = e^{+...})."""
    k, a = 37, 0.7
    Z = np.array([[np.exp(1j * a)]])
    y = oracle.idft(Z, k, M)[0]
    r = np.arange(M)
    assert np.max(np.abs(y - 2 * np.cos(2 * np.pi * k * r / M + a))) < 1e-12


# ------------------------------------------------------------------ O6 synthesis + round trips (P1, P2, P4, P5)
def test_synthesis_is_a_per_residue_fir(oracle, h):
    rng = np.random.default_rng(5)
    nq = 20
    y = rng.standard_normal((nq + P - 1, M))
    out = oracle.synthesis(y, h, M, P).reshape(nq, M)
    g = M * h.reshape(P, M)
    for r in (0, 1, 377, 1023):
        ref = np.convolve(y[:, r], g[:, r])[P - 1:P - 1 + nq]     # numpy's convolution, tap t on y[q-t]
        assert np.max(np.abs(out[:, r] - ref)) < 1e-12


def test_roundtrip_white_noise_error_bound_P1(oracle, h):
    rng = np.random.default_rng(1)
    T = 40
    x = rng.standard_normal((T + P - 1) * M)
    xh = roundtrip(oracle, x, h)
    sl = slice(16 * M, T * M)
    rel = np.linalg.norm(xh[sl] - x[sl]) / np.linalg.norm(x[sl])
    gain = np.dot(xh[sl], x[sl]) / np.dot(x[sl], x[sl])
    assert GOLD["P1_rel_l2"]["lo"] <= rel <= GOLD["P1_rel_l2"]["hi"]
    assert abs(gain - GOLD["P1_gain"]["value"]) < GOLD["P1_gain"]["tol"]


def test_roundtrip_tone_unit_gain_P2(oracle, h):
    T = 40
    n = np.arange((T + P - 1) * M)
    sl = slice(16 * M, T * M)
    x = np.cos(2 * np.pi * 300 * n / M + 0.3)
    xh = roundtrip(oracle, x, h)
    assert np.linalg.norm(xh[sl] - x[sl]) / np.linalg.norm(x[sl]) < GOLD["P2_tone_centre_err"]["hi"]
    x = np.cos(2 * np.pi * 300.25 * n / M + 0.3)
    xh = roundtrip(oracle, x, h)
    assert np.linalg.norm(xh[sl] - x[sl]) / np.linalg.norm(x[sl]) < 1e-4
    x = np.cos(2 * np.pi * 300.5 * n / M)
    xh = roundtrip(oracle, x, h)
    amp = math.sqrt(2.0 * np.mean(xh[sl] ** 2))
    assert abs(amp - GOLD["P2_tone_edge_amp"]["value"]) < GOLD["P2_tone_edge_amp"]["tol"]


def test_roundtrip_impulse_echoes_P4(oracle, h):
    T = 40
    x = np.zeros((T + P - 1) * M)
    n0 = 20 * M + 377
    x[n0] = 1.0
    xh = roundtrip(oracle, x, h)
    g = GOLD["P4_impulse_r377"]
    assert abs(xh[n0] - g["main"]) < g["tol"]                    # zero net delay (reading O6)
    for d, key in ((1, "echo1"), (2, "echo2"), (3, "echo3")):
        assert abs(xh[n0 + d * M] - g[key]) < g["tol"]
        assert abs(xh[n0 - d * M] - g[key]) < g["tol"]


@pytest.mark.parametrize("m,p,seed", [(8, 2, 0), (8, 3, 1), (8, 4, 2), (16, 2, 3)])
def test_whole_chain_brute_force_P5(oracle, m, p, seed):
    """O1 -> select -> O5 -> O6 equals one explicit double sum
       xhat[n] = sum_n' x[n'] * sum_q M h[n - qM] h[n' - qM] * Dir(n - n'),
       Dir(d) = [0 in sel] + 2 sum_{k in sel, k>=1} cos(2 pi k d / M)
    (written with a dense analysis matrix here, independent of the oracle's loops)."""
    rng = np.random.default_rng(seed)
    hh = oracle.prototype(m, p, 4.0)
    T = 9
    x = rng.standard_normal((T + p - 1) * m)
    k0 = int(rng.integers(0, m // 2 - 1))
    K = int(rng.integers(1, m // 2 - k0 + 1))
    got = roundtrip(oracle, x, hh, m, p, k0, K)
    # direct-form analysis from the oracle itself must agree with the folded form used above
    Yd = oracle.ppf_analysis(x, hh, m, p, T)
    assert np.max(np.abs(Yd - synth.station_ppf(x, T, m, p, hh))) < 1e-13
    L = m * p
    N = T * m
    want = np.zeros(N)
    sel = range(k0, k0 + K)
    for n in range(N):
        q, r = divmod(n, m)
        acc = 0.0
        for t in range(p):                       # slice q-t contributes through tap t
            mm = q - t
            if mm < 0:
                continue
            for j in range(L):                   # analysis of slice mm: sample mm*M + j, residue j % M
                d = (r - j)                      # e^{+2 pi i k r/M} e^{-2 pi i k j/M}
                dirk = sum((1.0 if k == 0 else 2.0 * math.cos(2 * math.pi * k * d / m)) for k in sel)
                acc += m * hh[r + t * m] * hh[j] * x[mm * m + j] * dirk
        want[n] = acc
    assert np.max(np.abs(got - want)) < 1e-12


# ------------------------------------------------------------------ O3/O4 tables and beamforming (P7)
def _rand_x(rng, S, K, T, dtype):
    lim = 100 if dtype == np.int8 else 20000
    return rng.integers(-lim, lim + 1, size=(S, 2, K, T, 2)).astype(dtype)


def test_tables_unit_modulus_and_formula(oracle):
    rng = np.random.default_rng(11)
    B, S, K, k0 = 3, 5, 7, 300
    tau = rng.uniform(-20e-9, 20e-9, (B, S))
    stec = np.array([5.0, 12.5])
    W, Dph = oracle.tables(tau, stec, K, k0)
    assert np.max(np.abs(np.abs(W) - 1)) < 1e-15 and np.max(np.abs(np.abs(Dph) - 1)) < 1e-15
    # exact rational arithmetic for the phase (fractions), then one cos/sin
    from fractions import Fraction
    for (b, s, j) in [(0, 0, 0), (2, 4, 6), (1, 3, 2)]:
        f = Fraction(100_000_000) + (k0 + j) * Fraction(200_000_000, 1024)
        turns = f * Fraction(tau[b, s])
        fr = float(turns - (turns.numerator // turns.denominator))
        assert abs(W[b, s, j] - complex(math.cos(2 * math.pi * fr), math.sin(2 * math.pi * fr))) < 1e-9
    for (d, j) in [(0, 0), (1, 6)]:
        f = Fraction(100_000_000) + (k0 + j) * Fraction(200_000_000, 1024)
        turns = Fraction(1_343_000_000) * Fraction(stec[d]) / f
        fr = float(turns - (turns.numerator // turns.denominator))
        assert abs(Dph[d, j] - complex(math.cos(2 * math.pi * fr), -math.sin(2 * math.pi * fr))) < 1e-9
    # dispersion applied (+phi) then removed (Dph) is the identity
    assert np.max(np.abs(Dph * np.conj(Dph) - 1)) < 1e-15


def test_dispersion_delay_sign_and_size(oracle):
    """Group delay -(1/2 pi) d(phase)/df of the *applied* dispersion e^{+i phi(f)} must be
    +1.343e9*STEC/f^2 seconds (larger at low f); the oracle's Dph is its conjugate."""
    stec = np.array([10.0])
    K, k0 = 200, 100
    _, Dph = oracle.tables(np.zeros((1, 1)), stec, K, k0)
    f = 100e6 + (k0 + np.arange(K)) * 200e6 / 1024
    ph = np.unwrap(np.angle(np.conj(Dph[0])))            # + phi(f)
    tg = -np.diff(ph) / (2 * np.pi * np.diff(f))
    fm = 0.5 * (f[1:] + f[:-1])
    assert np.allclose(tg, 1.343e9 * 10.0 / fm ** 2, rtol=1e-4)
    assert tg[0] > tg[-1] > 0


@pytest.mark.parametrize("dtype", [np.int8, np.int16])
def test_beamform_zero_delay_zero_stec_is_integer_sum(oracle, dtype):
    rng = np.random.default_rng(12)
    S, K, T = 4, 5, 6
    X = _rand_x(rng, S, K, T, dtype)
    X[0, 0, 0, 0] = (np.iinfo(dtype).min, np.iinfo(dtype).max)   # extreme values are legal input
    W, Dph = oracle.tables(np.zeros((2, S)), np.array([0.0]), K, 40)
    Z = oracle.beamform(X, W, Dph)
    ref = X.astype(np.int64).sum(axis=(0, 1))                    # [K][T][2]
    assert np.array_equal(Z[0].real, ref[..., 0]) and np.array_equal(Z[0].imag, ref[..., 1])
    assert np.array_equal(Z[1], Z[0])


def test_beamform_equals_einsum_and_window(oracle):
    rng = np.random.default_rng(13)
    S, B, D, K, T = 5, 3, 2, 6, 9
    X = _rand_x(rng, S, K, T, np.int16)
    tau = rng.uniform(-15e-9, 15e-9, (B, S))
    W, Dph = oracle.tables(tau, np.array([7.0, 11.0]), K, 123)
    Z = oracle.beamform(X, W, Dph)
    Xc = X[..., 0].astype(float) + 1j * X[..., 1]
    ref = np.einsum("dk,bsk,spkt->bdkt", Dph, W, Xc).reshape(B * D, K, T)
    assert np.max(np.abs(Z - ref)) < 1e-9
    Zw = oracle.beamform(X, W, Dph, 2, 4)
    assert np.array_equal(Zw, Z[:, :, 2:6])
    # transposed-operand guard: W[b][s] is not W[s][b]
    assert np.max(np.abs(Z - np.einsum("dk,sbk,spkt->bdkt", Dph, W[:, :3, :][:3].transpose(1, 0, 2)[:3][:, :3],
                                       Xc[:3]).reshape(B * D, K, T))) > 1.0


def test_coherent_gain_A6(oracle):
    """(i) matched phases: |Z|^2 = (2S a)^2 exactly; (ii) noise: Var = 2S sigma^2;
    (iii) off-axis array factor ~ S (two pols of a station add coherently in any direction)."""
    rng = np.random.default_rng(14)
    S, K, T, k0 = 24, 4, 4000, 300
    pos = synth.station_positions(S, 5)
    off = np.deg2rad(np.array([[0.0, 0.0], [0.2, 0.1]]))
    tau = synth.delays(pos, np.concatenate([off, off + np.deg2rad(2.0)]))[:3]
    W, Dph = oracle.tables(tau, np.array([0.0]), K, k0)
    a = 50.0
    # source in beam 1's direction: station phase = conj(W[1])
    sig = a * np.conj(W[1])[:, None, :, None] * np.ones((S, 2, K, 8))
    X = np.stack([np.rint(sig.real), np.rint(sig.imag)], axis=-1).astype(np.int16)
    Z = oracle.beamform(X, W, Dph)
    on = np.abs(Z[1]) ** 2
    assert np.allclose(on, (2 * S * a) ** 2, rtol=0.03)          # rounding of a*e^{i theta} to ints
    off_axis = np.mean(np.abs(Z[2]) ** 2)
    assert off_axis < on.mean() / 6                              # ~1/S on average for random geometry
    Xn = np.rint(rng.normal(0, 16.0, (S, 2, K, T, 2))).astype(np.int16)
    Zn = oracle.beamform(Xn, W, Dph)
    var_in = Xn.astype(float).var()
    assert abs(np.mean(np.abs(Zn[0]) ** 2) / (2 * 2 * S * var_in) - 1) < 0.03


def test_single_station_is_a_phase_rotation(oracle):
    rng = np.random.default_rng(15)
    K, T = 3, 5
    X = _rand_x(rng, 1, K, T, np.int8)
    X[:, 1] = 0
    tau = np.array([[7e-9]])
    W, Dph = oracle.tables(tau, np.array([9.0]), K, 77)
    Z = oracle.beamform(X, W, Dph)[0]
    Xc = X[0, 0, ..., 0].astype(float) + 1j * X[0, 0, ..., 1]
    assert np.max(np.abs(np.abs(Z) - np.abs(Xc))) < 1e-12
    f = 100e6 + (77 + np.arange(K)) * 200e6 / 1024
    rot = np.exp(1j * (2 * np.pi * f * 7e-9 - 2 * np.pi * 1.343e9 * 9.0 / f))     # north_star's w
    assert np.max(np.abs(Z - rot[:, None] * Xc)) < 1e-6 * np.abs(Xc).max()


# ------------------------------------------------------------------ O7/O8 trigger
def test_envelope_and_sigma(oracle):
    rng = np.random.default_rng(16)
    x = rng.standard_normal(1000)
    env, sig = oracle.envelope(x, 1)
    assert np.array_equal(env, np.abs(x))
    assert abs(sig - math.sqrt(np.mean(x ** 2))) < 1e-14
    lead = rng.standard_normal(7)
    env8, sig8 = oracle.envelope(x, 8, lead)
    xl = np.concatenate([lead, x])
    ref = np.sqrt(np.array([np.mean(xl[n:n + 8] ** 2) for n in range(1000)]))      # window n-7..n
    assert np.max(np.abs(env8 - ref)) < 1e-14
    assert abs(sig8 - math.sqrt(np.mean(ref ** 2))) < 1e-14


def test_candidates_best_trial_and_strictness(oracle):
    env = np.array([[1.0, 6.0, 2.0, 6.0, 12.0, 0.0],
                    [1.0, 14.0, 2.0, 5.0, 6.0, 0.0]])
    sigma = np.array([1.0, 2.0])                     # snr: [1,6,2,6,12,0] and [.5,7,1,2.5,3,0]
    smp, trl, cnt = oracle.candidates(env, sigma, 6.0)
    assert cnt == 2 and smp.tolist() == [1, 4] and trl.tolist() == [1, 0]   # n=1: trial 1 wins (7>6); n=3: 6 > 6 false
    smp, trl, cnt = oracle.candidates(env[:1], sigma[:1], 5.999)
    assert smp.tolist() == [1, 3, 4] and trl.tolist() == [0, 0, 0]
    # exact tie between trials -> lowest d
    smp, trl, cnt = oracle.candidates(np.array([[8.0], [16.0]]), sigma, 6.0)
    assert trl.tolist() == [0]
    # capacity: true count returned, first `cap` in order stored
    smp, trl, cnt = oracle.candidates(np.full((1, 10), 9.0), np.array([1.0]), 6.0, cap=4)
    assert cnt == 10 and smp.tolist() == [0, 1, 2, 3]


# ------------------------------------------------------------------ whole pipeline: P8, P9, P10
def _small_pipeline(oracle, w, **kw):
    _, _, tau = synth.geometry(w)
    return oracle.OraclePipeline(tau=tau, stec=np.array(w.stec), K=w.K, k0=w.k0, kappa=w.kappa, **kw), tau


def test_noise_level_closed_form_P8(oracle):
    w = synth.small(S=6, B=1, K=64, k0=200, T=48, n_pulses=0, sigma_in=4.0)
    pipe, tau = _small_pipeline(oracle, w)
    X = synth.generate_block(w, 0, tau=tau)
    series, sigma, _, _ = pipe.run_block(X)
    var_in = X.astype(float).var()
    closed = GOLD["P3_energy_mean"]["value"] * 4 * w.K * 2 * w.S * var_in
    meas = np.mean(series[0, 16 * M:] ** 2)
    assert abs(meas / closed - 1) < 0.03


def test_streaming_equals_one_shot_P9(oracle):
    w = synth.small(S=3, B=2, K=12, k0=40, T=40, n_pulses=1, stec=(10.0, 12.0))
    pipe, tau = _small_pipeline(oracle, w)
    X = synth.generate_block(w, 0, tau=tau)
    whole, _, _, _ = pipe.run_block(X)
    pipe.reset()
    parts = []
    offs = []
    for a, b in ((0, 8), (8, 24), (24, 40)):
        offs.append(pipe.offset)
        s, _, _, _ = pipe.run_block(np.ascontiguousarray(X[:, :, :, a:b]))
        parts.append(s)
    assert offs == [0, 8 * M, 24 * M]
    assert np.array_equal(np.concatenate(parts, axis=1), whole)          # bit-identical
    # windowed evaluation (used for sampled parity at full size) is the same numbers
    win = pipe.series_window(X, 3, 20, 5)
    assert np.array_equal(win, whole[3, 20 * M:25 * M])
    win0 = pipe.series_window(X, 1, 0, 4)
    assert np.array_equal(win0, whole[1, :4 * M])


def test_pulse_recovered_at_injected_sample_P10(oracle):
    """Physics pin for the signs of tau and phi (readings A3, A9): a pulse injected from beam 0's
    direction with STEC 10 is recovered by beam 0 at the injected sample with >= 0.75 of the ideal
    band-limited peak, fires the trigger there, and is much weaker with the wrong dispersion sign,
    without de-dispersion, or in a beam 0.2 degrees away is not boosted."""
    w = synth.small(S=6, B=2, K=244, k0=256, T=96, n_pulses=1, sigma_in=6.0, dtype="ci16", kappa=6.0)
    pos, off, tau = synth.geometry(w)
    tau = synth.delays(pos, np.deg2rad(np.array([[0.0, 0.0], [0.2, 0.0]])))
    X = synth.generate_block(w, 0, tau=tau)
    pl = synth.make_pulses(w)[0]
    assert pl.beam in (0, 1)
    n_inj = int(round(pl.sample))
    pipe = oracle.OraclePipeline(tau=tau, stec=np.array([10.0]), K=w.K, k0=w.k0, kappa=6.0)
    series, sigma, cands, total = pipe.run_block(X)
    b = pl.beam
    peak_n = int(np.argmax(np.abs(series[b])))
    assert abs(peak_n - n_inj) <= 1
    ideal = 2 * w.S * pl.amp
    assert 0.75 * ideal < abs(series[b, peak_n]) < 1.05 * ideal + 5 * sigma[b]
    assert any(c.series == b and abs(c.sample - n_inj) <= 1 for c in cands)
    assert np.max(np.abs(series[1 - b])) < 0.6 * abs(series[b, peak_n])
    for bad in (-10.0, 0.0):
        p2 = oracle.OraclePipeline(tau=tau, stec=np.array([bad]), K=w.K, k0=w.k0, kappa=6.0)
        s2, _, _, _ = p2.run_block(X)
        assert np.max(np.abs(s2[b])) < 0.6 * abs(series[b, peak_n])
    # wrong sign of the geometric delays loses the coherent sum too
    p3 = oracle.OraclePipeline(tau=-tau, stec=np.array([10.0]), K=w.K, k0=w.k0, kappa=6.0)
    s3, _, _, _ = p3.run_block(X)
    assert np.max(np.abs(s3[b])) < 0.6 * abs(series[b, peak_n])


def test_config0_timedomain_generator_small(oracle):
    """The config-0 recipe (full time-domain path through the station PPF) at a reduced T:
    oracle reconstruction finds the injected pulse at the right sample."""
    from dataclasses import replace
    w = replace(synth.config(0), T=64, index=0)
    pos, off, tau = synth.geometry(w)
    X = synth.generate_block(w, 0, tau=tau)
    assert X.shape == (4, 2, 16, 64, 2) and X.dtype == np.int16
    assert abs(X.astype(float).std() - 8.0) < 1.0
    pl = synth.make_pulses(w)[0]
    pipe = oracle.OraclePipeline(tau=tau, stec=np.array(w.stec), K=w.K, k0=w.k0, kappa=5.0)
    series, sigma, cands, _ = pipe.run_block(X)
    n_inj = int(round(pl.sample))
    # 16 sub-bands = 3 MHz: the band-limited pulse is a ~64-sample wave packet with a 3.4-sample
    # carrier, so noise can move the largest lobe by one carrier period
    assert abs(int(np.argmax(np.abs(series[pl.beam]))) - n_inj) <= 4
    assert np.abs(series[pl.beam]).max() > 0.6 * 2 * w.S * pl.amp


def test_golden_values_are_regenerated_by_the_committed_script():
    """tests/golden/make_ppf_pins.py (numpy / scipy only, no oracle code) reproduces every stored number."""
    import importlib.util
    path = os.path.join(os.path.dirname(__file__), "golden", "make_ppf_pins.py")
    spec = importlib.util.spec_from_file_location("make_ppf_pins", path)
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    assert mod.main() == 0
