"""Pins of the oracle functions for the rows "next" of SURVEY.md 8(f) (O9..O13), against things other than
themselves: a library routine run on the same system (scipy.sparse.linalg.lsmr), dense least squares,
the invariants the algorithm guarantees, closed forms, brute force on tiny sizes, hand-worked tables and
the physics of the generator.  No GPU, no CUDA library."""
import numpy as np
import pytest

from paper_1612_06592_b200 import synth

M, P = 1024, 16


@pytest.fixture(scope="module")
def h(oracle):
    return oracle.prototype(M, P, 9.0)


def _analysed(oracle, h_, T, seed, M_=M, P_=P, k0=0, K=None):
    rng = np.random.default_rng(seed)
    x = rng.standard_normal((T + P_ - 1) * M_)
    Y = synth.station_ppf(x, T, M_, P_, h_)
    K = M_ // 2 - k0 if K is None else K
    Z = np.ascontiguousarray(Y[:, k0:k0 + K].T)
    y = oracle.idft(Z, k0, M_)
    return x, np.concatenate([np.zeros((P_ - 1, M_)), y])


# ------------------------------------------------------------------ O11 LSMR inversion (f1)
def test_lsmr_equals_scipy_lsmr_on_the_same_system(oracle, h):
    """The recurrences, iterate by iterate, are those of a library LSMR (scipy) run on the dense FIR system of
    one residue with no damping and no stopping test."""
    from scipy.sparse.linalg import lsmr
    T = 40
    _, ylead = _analysed(oracle, h, T, 11)
    for iters in (1, 2, 7, 25):
        got = oracle.lsmr_inversion(ylead, h, iters).reshape(T, M)
        for r in (0, 1, 377, 511, 512, 1023):
            A = oracle.ppf_system(h, r, T + P - 1)
            xs = lsmr(A, ylead[:, r] / M, damp=0.0, atol=0.0, btol=0.0, conlim=0.0, maxiter=iters)[0]
            assert np.max(np.abs(xs[P - 1:P - 1 + T] - got[:, r])) < 1e-12 * max(1.0, np.abs(xs).max()), (iters, r)


@pytest.mark.parametrize("Ms,Ps", [(8, 2), (8, 3), (8, 4), (16, 4)])
def test_lsmr_converges_to_the_minimum_norm_least_squares_solution(oracle, Ms, Ps):
    """Small sizes: after many iterations the result is numpy.linalg.lstsq's (minimum-norm) solution of the dense
    system; the system matrix itself is pinned against the analysis definition O1 (y/M = H x exactly when every
    bin, Nyquist included, is kept)."""
    hs = oracle.prototype(Ms, Ps, 9.0)
    T = 12
    rng = np.random.default_rng(5)
    x = rng.standard_normal((T + Ps - 1) * Ms)
    # O1 fold (all M bins): u[m][r] = sum_t h[r + t M] x[(m + t) M + r] = (H x)[m]
    u = np.zeros((T, Ms))
    for t in range(Ps):
        u += hs.reshape(Ps, Ms)[t][None, :] * x.reshape(T + Ps - 1, Ms)[t:t + T]
    for r in range(Ms):
        A = oracle.ppf_system(hs, r, T, Ms, Ps)
        assert np.allclose(A @ x.reshape(-1, Ms)[:, r], u[:, r], atol=1e-14)
    ylead = np.concatenate([np.zeros((Ps - 1, Ms)), Ms * u])
    got = oracle.lsmr_inversion(ylead, hs, 400, Ms, Ps).reshape(T, Ms)
    for r in range(Ms):
        A = oracle.ppf_system(hs, r, T + Ps - 1, Ms, Ps)
        ref = np.linalg.lstsq(A, ylead[:, r] / Ms, rcond=None)[0]
        assert np.max(np.abs(ref[Ps - 1:Ps - 1 + T] - got[:, r])) < 1e-8, r


def test_lsmr_residual_decreases_and_beats_the_matched_filter(oracle, h):
    """||r_k|| = ||H x_k - y|| is non-increasing in k (a property LSMR guarantees), and the paper's reason for
    LSMR: the reconstruction error of white noise (pin P1: 0.19 for the matched synthesis) falls below 0.06
    after 25 iterations ("convergence ... after approximately 25 iterations")."""
    T = 72
    x, ylead = _analysed(oracle, h, T, 3)
    taps = h.reshape(P, M)
    prev = None
    for k in (1, 2, 3, 5, 8, 13, 25):
        xk = oracle.lsmr_inversion(ylead, h, k).reshape(T, M)
        # residual on the interior equations whose 16 unknowns all lie inside the output
        res = np.zeros((T - P + 1, M))
        for t in range(P):
            res += taps[t][None, :] * xk[t:t + T - P + 1]
        res -= ylead[P - 1:P - 1 + T - P + 1] / M
        nrm = np.linalg.norm(res[16:-16])
        if prev is not None:
            assert nrm <= prev * (1 + 1e-9), k
        prev = nrm
    x25 = oracle.lsmr_inversion(ylead, h, 25)
    xm = oracle.synthesis(ylead, h)
    ref = x[:T * M]
    sl = slice(20 * M, (T - 20) * M)
    e_lsmr = np.linalg.norm(x25[sl] - ref[sl]) / np.linalg.norm(ref[sl])
    e_matched = np.linalg.norm(xm[sl] - ref[sl]) / np.linalg.norm(ref[sl])
    assert 0.17 < e_matched < 0.21 and e_lsmr < 0.06


def test_lsmr_one_iteration_is_the_scaled_matched_filter(oracle, h):
    """Special case: x_1 is proportional to H^T y per residue, i.e. to O6's output (reading A8: the matched
    synthesis is LSMR's first step)."""
    T = 30
    _, ylead = _analysed(oracle, h, T, 9)
    x1 = oracle.lsmr_inversion(ylead, h, 1).reshape(T, M)
    xm = oracle.synthesis(ylead, h).reshape(T, M)
    for r in (3, 400, 777):
        a, b = x1[:, r], xm[:, r]
        c = (a @ b) / (b @ b)
        assert np.linalg.norm(a - c * b) < 1e-10 * np.linalg.norm(a) and c > 0


# ------------------------------------------------------------------ O12 exact de-dispersion (f2)
def _bandlimited(rng, n, M_, k_lo, k_hi):
    X = np.fft.rfft(rng.standard_normal(n))
    kf = np.arange(X.size) * M_ / n
    X[(kf < k_lo) | (kf >= k_hi)] = 0
    return np.fft.irfft(X, n)


def test_dedisperse_factor_properties(oracle):
    D = oracle.dedisperse_factor(12.0, 16384)
    assert D.size == 8193
    assert np.max(np.abs(np.abs(D[1:-1]) - 1.0)) < 1e-14
    assert D[0].imag == 0 and D[-1].imag == 0
    # the phase is the dispersion law at the bin's sky frequency, exact in rational arithmetic
    from fractions import Fraction
    for j in (1, 1000, 8191):
        f = Fraction(100_000_000) + Fraction(j) * Fraction(200_000_000, 16384)
        turns = float((Fraction(1343_000_000) * 12 / f) % 1)
        assert abs(D[j] - np.exp(-2j * np.pi * turns)) < 1e-9
    # group delay -(1/2 pi) d(arg D)/df is negative: de-dispersion advances the low frequencies (reading A3)
    j = 2000
    dphi = np.angle(D[j + 1] * np.conj(D[j]))
    assert dphi > 0


def test_dedisperse_zero_stec_is_a_one_slice_delay(oracle):
    rng = np.random.default_rng(1)
    T = 37
    x = rng.standard_normal((T + 2) * M)
    y = oracle.dedisperse_exact(x, 0.0)
    assert y.size == T * M
    assert np.max(np.abs(y - x[M:M + T * M])) < 1e-12


@pytest.mark.parametrize("stec,tol", [(5.0, 1e-3), (12.0, 2e-3), (20.0, 4e-3)])
def test_dispersion_applied_then_removed_is_the_identity(oracle, stec, tol):
    """north_star: "dispersion phase applied then removed giving the identity".  The dispersion is applied with ONE
    long transform over the whole signal (not the oracle's segmentation); the overlap-save result equals the
    undispersed signal, one slice late, up to the truncation of the chirp's tails by the one-slice guard."""
    rng = np.random.default_rng(2)
    T = 64
    n = (T + 2) * M
    x = _bandlimited(rng, n, M, 24, 511.5)
    j = np.arange(n // 2 + 1)
    f = 100e6 + j * (200e6 / n)
    Dl = np.exp(+2j * np.pi * np.mod(1.343e9 * stec / f, 1.0))
    Dl[0] = Dl[0].real
    Dl[-1] = Dl[-1].real
    xd = np.fft.irfft(np.fft.rfft(x) * Dl, n)
    y = oracle.dedisperse_exact(xd, stec)
    ref = x[M:M + T * M]
    sl = slice(4 * M, (T - 4) * M)
    assert np.linalg.norm(y[sl] - ref[sl]) / np.linalg.norm(ref[sl]) < tol
    # and it is not a no-op: without de-dispersion the dispersed signal is far from the original
    assert np.linalg.norm(xd[M:M + T * M][sl] - ref[sl]) / np.linalg.norm(ref[sl]) > 0.5


def test_dedisperse_segment_equals_direct_circular_convolution(oracle):
    """Brute force on a small size (M = 8, segment = 128 samples): the rfft * D * irfft step is the circular
    convolution with d = irfft(D), written as a double loop."""
    Ms = 8
    rng = np.random.default_rng(3)
    T = 14                                            # exactly one segment: 16 slices in, 14 out
    x = rng.standard_normal((T + 2) * Ms)
    y = oracle.dedisperse_exact(x, 7.0, M=Ms, clock_hz=200e6, f_zone_hz=100e6)
    nfft = 16 * Ms
    d = np.fft.irfft(oracle.dedisperse_factor(7.0, nfft), nfft)
    full = np.zeros(nfft)
    for n in range(nfft):
        for m in range(nfft):
            full[n] += d[(n - m) % nfft] * x[m]
    assert np.max(np.abs(y - full[Ms:Ms + T * Ms])) < 1e-12


def test_exact_dedispersion_recovers_more_of_a_pulse_than_the_subband_staircase(oracle, h):
    """Physics (reading A9): the per-sub-band phase costs a few per cent of the pulse amplitude; the exact form
    does not.  One noiseless dispersed pulse through the whole chain, both ways."""
    w = synth.small(S=1, B=1, K=488, k0=24, T=64, dtype="ci16", sigma_in=0.0, stec=(12.0,), pulse_stec=12.0,
                    n_pulses=1, kappa=6.0)
    tau = np.zeros((1, 1))
    pulse = synth.Pulse(0, 30 * M + 517.25, 12.0, 2000.0)
    m0, F = synth.pulse_footprint(w, pulse, tau[0], 48)
    Z = np.zeros((w.K, w.T), dtype=np.complex128)
    Z[:, m0:m0 + F.shape[2]] = F[0]
    Xs = np.zeros((1, 2, w.K, w.T, 2), dtype=np.int16)
    Xs[0, 0, :, :, 0] = np.rint(Z.real)
    Xs[0, 0, :, :, 1] = np.rint(Z.imag)
    sub = oracle.OraclePipeline(tau=tau, stec=np.array([12.0]), K=w.K, k0=w.k0)
    ex = oracle.OraclePipeline(tau=tau, stec=np.array([12.0]), K=w.K, k0=w.k0, dedisp="exact")
    ys, _, _, _ = sub.run_block(Xs)
    ye, _, _, _ = ex.run_block(Xs)
    n_s = int(np.argmax(np.abs(ys[0])))
    n_e = int(np.argmax(np.abs(ye[0])))
    assert abs(n_s - 30 * M - 517) <= 1
    assert abs(n_e - M - 30 * M - 517) <= 1              # one slice late
    assert np.abs(ye[0]).max() > 1.01 * np.abs(ys[0]).max()
    # with the wrong sign of the phase the pulse is smeared out
    wrong = oracle.dedisperse_exact(np.concatenate([np.zeros(2 * M), oracle.OraclePipeline(
        tau=tau, stec=np.array([12.0]), K=w.K, k0=w.k0, dedisp="exact").run_block(Xs)[0][0]]), -24.0)
    assert np.abs(wrong).max() < 0.6 * np.abs(ye[0]).max()


# ------------------------------------------------------------------ O9 causal sigma, O10 clustering (f3)
def test_cluster_hand_worked_table(oracle):
    beam = [0, 0, 0, 0, 1, 1, 2, 2, 2]
    smp = [10, 12, 40, 41, 5, 105, 7, 8, 9]
    snr = [6.5, 7.0, 6.1, 6.1, 9.0, 6.2, 6.3, 8.0, 8.0]
    ev = oracle.cluster(beam, smp, snr, gap=10)
    assert [(e["beam"], e["first"], e["last"], e["count"], e["peak"]) for e in ev] == [
        (0, 10, 12, 2, 1),       # 10, 12 within the gap; peak = the larger snr
        (0, 40, 41, 2, 2),       # 12 -> 40 exceeds the gap; equal snr -> the lowest sample
        (1, 5, 5, 1, 4),         # a beam change always starts an event
        (1, 105, 105, 1, 5),
        (2, 7, 9, 3, 7),         # tie between samples 8 and 9 -> sample 8
    ]
    assert oracle.cluster([], [], [], 10) == []
    # gap is inclusive: a difference of exactly `gap` still joins
    assert len(oracle.cluster([0, 0], [0, 10], [7.0, 7.0], 10)) == 1
    assert len(oracle.cluster([0, 0], [0, 11], [7.0, 7.0], 10)) == 2


def test_causal_sigma_reference_and_equivalence_on_stationary_noise(oracle):
    """O9: block i is judged against sigma of block i-1 (block 0: sigma_init or itself).  On stationary noise
    the causal and the two-pass candidate sets agree except where the envelope is within the closed-form
    estimation error of sigma around the threshold: rel. std of an RMS over N_eff independent Gaussian samples
    = 1/sqrt(2 N_eff)."""
    w = synth.small(S=3, B=2, K=24, k0=100, T=64, dtype="ci8", n_pulses=0, blocks=3, kappa=3.5)
    _, _, tau = synth.geometry(w)
    blocks = [synth.generate_block(w, b, tau=tau) for b in range(3)]
    two = oracle.OraclePipeline(tau=tau, stec=np.asarray(w.stec), K=w.K, k0=w.k0, kappa=w.kappa)
    cau = oracle.OraclePipeline(tau=tau, stec=np.asarray(w.stec), K=w.K, k0=w.k0, kappa=w.kappa, sigma_mode="causal")
    N = w.T * 1024
    sig_hist = []
    for i, X in enumerate(blocks):
        s2, sig2, c2, n2 = two.run_block(X)
        s1, sig1, c1, n1 = cau.run_block(X)
        assert np.array_equal(s1, s2) and np.array_equal(sig1, sig2)        # the series and sigma are the same
        ref = sig2 if i == 0 else sig_hist[-1]
        assert np.array_equal(cau.last_sigma_ref, ref)
        assert all(c.sigma == ref[c.series] for c in c1)
        a = {(c.series, c.sample) for c in c1}
        b = {(c.series, c.sample) for c in c2}
        if i == 0:
            assert a == b
        # the series holds 2K of M real degrees of freedom per slice -> N_eff = N * 2K/M independent samples;
        # the difference of two independent RMS estimates has relative std sqrt(2) / sqrt(2 N_eff); 4 of those
        delta = 4.0 * np.sqrt(2.0) / np.sqrt(2.0 * N * (2.0 * w.K / 1024.0))
        for s, n in a ^ b:
            e = abs(s2[s, n - i * N]) / (w.kappa * sig2[s])
            assert abs(e - 1.0) < delta, (s, n, e)
        sig_hist.append(sig2)
    # sigma_init is used for block 0 when given
    init = np.array([10.0, 1e9])
    ini = oracle.OraclePipeline(tau=tau, stec=np.asarray(w.stec), K=w.K, k0=w.k0, kappa=w.kappa, sigma_mode="causal",
                                sigma_init=init)
    s0, _, c0, _ = ini.run_block(blocks[0])
    assert {c.series for c in c0} == {0}
    assert len(c0) == int((np.abs(s0[0]) > w.kappa * 10.0).sum())


# ------------------------------------------------------------------ O13 two-stage beamforming (f4)
def test_requantise_rounding_and_clipping(oracle):
    Z = np.array([0.5 + 1.5j, 2.5 - 0.5j, 1e9 - 1e9j, -0.49 + 0.51j])
    q = oracle.requantise(Z, 1.0)
    assert q.dtype == np.int16
    assert q.tolist() == [[0, 2], [2, 0], [32767, -32767], [0, 1]]          # ties to even, clip
    assert oracle.requantise(np.array([3.0 + 0j]), 0.5).tolist() == [[2, 0]]


def test_two_stage_beamforming_equals_single_stage_up_to_requantisation(oracle):
    """sub-arrays pre-beamformed on the first cluster, final beams on the second -- "the same linear
    sum split in two".  Stage 1 per sub-array g (its own stations, pointing centre beam), re-quantised to int16
    with a large scale, fed as pseudo-stations to stage 2; equals the one-stage sum to the rounding bound."""
    w = synth.small(S=6, B=3, K=8, k0=50, T=40, dtype="ci8", stec=(0.0,))
    _, _, tau = synth.geometry(w)
    X = synth.generate_block(w, 0, tau=tau)
    W, Dph = oracle.tables(tau, np.zeros(1), w.K, w.k0)
    Z1 = oracle.beamform(X, W, Dph)                                        # [B][K][T]
    groups = [(0, 1, 2), (3, 4, 5)]
    scale = 64.0
    Xs2 = np.zeros((len(groups), 2, w.K, w.T, 2), dtype=np.int16)
    tau1 = np.zeros((1, 3))
    for g, st in enumerate(groups):
        Wg, Dg = oracle.tables(tau1, np.zeros(1), w.K, w.k0)               # unit weights: sum of the sub-array
        Zg = oracle.beamform(np.ascontiguousarray(X[list(st)]), Wg, Dg)    # [1][K][T]
        Xs2[g, 0] = oracle.requantise(Zg[0], scale)                         # pseudo-station, second polarisation empty
    # exact only if the stage-2 weight is common to the stations of a group: use the group's mean delay
    tau2 = np.stack([tau[:, list(st)].mean(axis=1) for st in groups], axis=1)
    W2, D2 = oracle.tables(tau2, np.zeros(1), w.K, w.k0)
    Z2 = oracle.beamform(Xs2, W2, D2) / scale
    # reference: the same composite weights applied in one stage
    Wc = np.empty_like(W)
    for g, st in enumerate(groups):
        for s in st:
            Wc[:, s, :] = W2[:, g, :]
    Zc = oracle.beamform(X, Wc, Dph)
    bound = len(groups) * np.sqrt(0.5) / scale
    assert np.max(np.abs(Z2 - Zc)) <= bound * 1.0001
    # (the composite weights differ from the per-station ones: the beam-shape cost of the split, which the
    # paper leaves "under investigation", is not asserted here)
    assert Z1.shape == Zc.shape
