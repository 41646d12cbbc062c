"""GPU parity for the rows "next" of SURVEY.md 8(f), each against the oracle function pinned in
tests/test_oracle_next_pins.py: f3 (trigger-only mode, causal sigma, event clustering), f1 (LSMR inversion),
f2 (exact de-dispersion), f4 (two-stage beamforming)."""
import numpy as np
import pytest

from paper_1612_06592_b200 import binding, synth
from parity_util import GUARD, assert_close, check_candidates, oracle_snr

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch():
    import torch as t
    assert t.cuda.is_available(), "GPU tests need a CUDA device"
    binding.load()
    return t


def _blocks(w):
    _, _, tau = synth.geometry(w)
    return tau, [synth.generate_block(w, b, tau=tau) for b in range(w.blocks)]


def _run(torch, p, X, T, want_series=True):
    series, cand, count, sigma = binding.new_outputs(p, T)
    p.run_block(torch.from_numpy(X).cuda(), T, series if want_series else None, cand, count, sigma)
    torch.cuda.synchronize()
    return (series.cpu().numpy() if want_series else None, binding.candidates_to_numpy(cand, count),
            int(count.item()), sigma.cpu().numpy(), cand, count)


# ------------------------------------------------------------------------------------------ f3
TRIGGER_ONLY_CASES = [
    dict(S=4, B=3, K=24, k0=200, T=208, dtype="ci8", n_pulses=5, blocks=2, kappa=4.5),
    dict(S=4, B=2, K=16, k0=300, T=104, dtype="ci16", n_pulses=3, blocks=2, kappa=4.0),
    dict(S=6, B=3, K=33, k0=470, T=72, dtype="ci8", stec=(8.0, 10.0, 12.0, 14.0), n_pulses=3, blocks=2, kappa=4.0),
    dict(S=24, B=24, K=40, k0=100, T=136, dtype="ci8", n_pulses=4, blocks=2, kappa=4.5),
]


@pytest.mark.parametrize("kw", TRIGGER_ONLY_CASES)
def test_trigger_only_mode_equals_the_oracle(torch, oracle, kw):
    """series == NULL: no series in HBM, sigma and candidates as defined by O7/O8 -- the flagged
    chunks are recomputed from X after sigma is known.  Two blocks (carried history at a flagged first step),
    several scratch chunks, D = 1 and D > 1 (best trial per sample)."""
    w = synth.small(**kw)
    tau, blocks = _blocks(w)
    pipe = oracle.OraclePipeline(tau=tau, stec=np.asarray(w.stec), K=w.K, k0=w.k0, kappa=w.kappa)
    p = binding.plan_for(w, tau)
    p.set_trigger(w.kappa, 1, 1 << 16)
    p.set_scratch_limit(w.B * w.K * 8 * 64)           # three or four chunks per block
    full = binding.plan_for(w, tau)
    full.set_trigger(w.kappa, 1, 1 << 16)
    offset = 0
    for X in blocks:
        ref, sig_ref, _, _ = pipe.run_block(X)
        _, rec, n, sigma, _, _ = _run(torch, p, X, w.T, want_series=False)
        np.testing.assert_allclose(sigma, sig_ref, rtol=5e-6)
        env, sig = oracle_snr(oracle, ref, 1)
        ndef, _ = check_candidates(rec, n, env, sig, w.B, w.D, w.kappa, offset)
        assert ndef > 0
        # and the list is the one the series path reports (up to the guard band)
        _, rec_f, n_f, _, _, _ = _run(torch, full, X, w.T)
        a = {(int(r["series"]) // w.D, int(r["sample"])) for r in rec}
        b = {(int(r["series"]) // w.D, int(r["sample"])) for r in rec_f}
        for bm, smp in a ^ b:
            e = (env[bm * w.D:(bm + 1) * w.D, smp - offset] / sig[bm * w.D:(bm + 1) * w.D]).max() / w.kappa
            assert abs(e - 1.0) <= GUARD
        offset += w.T * 1024
    p.destroy()
    full.destroy()


@pytest.mark.parametrize("with_series", [True, False])
@pytest.mark.parametrize("kw", [
    dict(S=4, B=3, K=24, k0=200, T=96, dtype="ci8", n_pulses=6, blocks=4, kappa=4.5),
    dict(S=6, B=2, K=33, k0=470, T=72, dtype="ci8", stec=(8.0, 10.0, 12.0), n_pulses=4, blocks=3, kappa=4.0),
])
def test_causal_sigma_parity(torch, oracle, kw, with_series):
    """LOFAR_SIGMA_CAUSAL: block i against sigma of block i-1 (O9); block 0 against itself.  Candidates come out of
    the inverse-PPF epilogue (from block 1 on), with and without a series in HBM."""
    w = synth.small(**kw)
    tau, blocks = _blocks(w)
    pipe = oracle.OraclePipeline(tau=tau, stec=np.asarray(w.stec), K=w.K, k0=w.k0, kappa=w.kappa, sigma_mode="causal")
    p = binding.plan_for(w, tau)
    p.set_trigger(w.kappa, 1, 1 << 16)
    p.set_sigma_mode(binding.LOFAR_SIGMA_CAUSAL)
    offset = 0
    for i, X in enumerate(blocks):
        ref, sig_ref, _, _ = pipe.run_block(X)
        got, rec, n, sigma, _, _ = _run(torch, p, X, w.T, want_series=with_series)
        np.testing.assert_allclose(sigma, sig_ref, rtol=5e-6)
        if with_series:
            for s in range(w.nseries):
                assert_close(got[s], ref[s], f"block {i} series {s}")
        env, _ = oracle_snr(oracle, ref, 1)
        check_candidates(rec, n, env, pipe.last_sigma_ref, w.B, w.D, w.kappa, offset)
        offset += w.T * 1024
    # checkpoint in the middle of the stream: the reference level travels with the state
    q = binding.plan_for(w, tau)
    q.set_trigger(w.kappa, 1, 1 << 16)
    q.set_sigma_mode(binding.LOFAR_SIGMA_CAUSAL)
    q.set_state(p.get_state())
    X = synth.generate_block(w, w.blocks, tau=tau)
    _, rec_p, n_p, _, _, _ = _run(torch, p, X, w.T, want_series=with_series)
    _, rec_q, n_q, _, _, _ = _run(torch, q, X, w.T, want_series=with_series)
    assert n_p == n_q and np.array_equal(rec_p, rec_q)
    p.destroy()
    q.destroy()


def test_causal_sigma_init_and_streaming(torch, oracle):
    """sigma_init_host gives block 0 its level; the same through lofar_stream_push without a series."""
    w = synth.small(S=4, B=3, K=24, k0=200, T=64, dtype="ci8", n_pulses=4, blocks=3, kappa=4.5)
    tau, blocks = _blocks(w)
    init = np.full(w.nseries, 1.05 * np.sqrt(0.9341 * 4 * w.K * 2 * w.S) * w.sigma_in)
    pipe = oracle.OraclePipeline(tau=tau, stec=np.asarray(w.stec), K=w.K, k0=w.k0, kappa=w.kappa, sigma_mode="causal",
                                 sigma_init=init)
    p = binding.plan_for(w, tau)
    p.set_trigger(w.kappa, 1, 8192)
    p.set_sigma_mode(binding.LOFAR_SIGMA_CAUSAL, init)
    p.stream_reset()
    outs = []
    for X in blocks:
        cand_h = torch.zeros((8192, 24), dtype=torch.uint8).pin_memory()
        count_h = torch.zeros(1, dtype=torch.int32).pin_memory()
        sigma_h = torch.zeros(w.nseries, dtype=torch.float32).pin_memory()
        Xh = torch.from_numpy(X).pin_memory()
        p.stream_push(Xh, w.T, None, cand_h, count_h, sigma_h)
        outs.append((Xh, cand_h, count_h, sigma_h))
    p.stream_sync()
    offset = 0
    for X, (_, cand_h, count_h, sigma_h) in zip(blocks, outs):
        ref, sig_ref, _, _ = pipe.run_block(X)
        np.testing.assert_allclose(sigma_h.numpy(), sig_ref, rtol=5e-6)
        env, _ = oracle_snr(oracle, ref, 1)
        rec = binding.candidates_to_numpy(cand_h.numpy(), int(count_h.item()))
        check_candidates(rec, int(count_h.item()), env, np.asarray(pipe.last_sigma_ref, dtype=np.float64), w.B, w.D,
                         w.kappa, offset)
        offset += w.T * 1024
    p.destroy()


def test_cluster_parity(torch, oracle):
    """lofar_cluster on the candidate list of a block with pulses (several candidates per pulse) and on a hand-built
    list, against O10."""
    w = synth.small(S=6, B=4, K=33, k0=470, T=96, dtype="ci8", stec=(8.0, 10.0, 12.0), n_pulses=6, kappa=3.6)
    tau, blocks = _blocks(w)
    p = binding.plan_for(w, tau)
    p.set_trigger(w.kappa, 1, 1 << 16)
    _, rec, n, sigma, cand, count = _run(torch, p, blocks[0], w.T)
    assert n > 50
    for gap in (0, 3, 64, 5000):
        events = torch.zeros((4096, 48), dtype=torch.uint8, device="cuda")
        nev = torch.zeros(1, dtype=torch.int32, device="cuda")
        p.cluster(cand, count, gap, events, nev)
        torch.cuda.synchronize()
        ev = binding.events_to_numpy(events, nev)
        snr = rec["env"].astype(np.float64) / rec["sigma"].astype(np.float64)
        want = oracle.cluster(rec["series"] // w.D, rec["sample"].astype(np.int64), snr, gap)
        assert int(nev.item()) == len(want) == ev.size
        for e, o in zip(ev, want):
            assert (int(e["beam"]), int(e["first_sample"]), int(e["last_sample"]), int(e["count"])) == \
                   (o["beam"], o["first"], o["last"], o["count"])
            pk = rec[o["peak"]]
            if int(e["peak_sample"]) != int(pk["sample"]):        # fp32 vs fp64 ratio: only an exact-tie class may differ
                assert abs(e["peak_snr"] - snr[o["peak"]]) <= 1e-6 * snr[o["peak"]]
            else:
                assert int(e["peak_trial"]) == int(pk["trial"]) and e["peak_env"] == pk["env"]
                assert abs(e["peak_snr"] - snr[o["peak"]]) <= 1e-6 * snr[o["peak"]]
        if gap == 0:
            assert len(want) == n or any(o["count"] > 1 for o in want) is False
    # hand-built list (the oracle pin's table) through the same call
    beam = np.array([0, 0, 0, 0, 1, 1, 2, 2, 2])
    smp = np.array([10, 12, 40, 41, 5, 105, 7, 8, 9])
    s = np.array([6.5, 7.0, 6.1, 6.1, 9.0, 6.2, 6.3, 8.0, 8.0], dtype=np.float32)
    raw = np.zeros(9, dtype=binding.CANDIDATE_DTYPE)
    raw["series"] = beam * w.D
    raw["sample"] = smp
    raw["env"] = s
    raw["sigma"] = 1.0
    cd = torch.from_numpy(raw.view(np.uint8).reshape(9, 24).copy()).cuda()
    cn = torch.tensor([9], dtype=torch.int32, device="cuda")
    events = torch.zeros((16, 48), dtype=torch.uint8, device="cuda")
    nev = torch.zeros(1, dtype=torch.int32, device="cuda")
    p.cluster(cd, cn, 10, events, nev)
    torch.cuda.synchronize()
    ev = binding.events_to_numpy(events, nev)
    assert [(int(e["beam"]), int(e["first_sample"]), int(e["last_sample"]), int(e["count"]), int(e["peak_sample"]))
            for e in ev] == [(0, 10, 12, 2, 12), (0, 40, 41, 2, 40), (1, 5, 5, 1, 5), (1, 105, 105, 1, 105),
                             (2, 7, 9, 3, 8)]
    p.destroy()


# ------------------------------------------------------------------------------------------ f1
LSMR_TOL = dict(rel=2e-5, mx=2e-4)     # fp32 vectors through 25 iterations (f1): twice north_star's


def _close(got, ref, what, rel, mx):
    got = np.asarray(got, dtype=np.float64)
    nrm = np.linalg.norm(ref)
    rms = nrm / np.sqrt(ref.size)
    err = np.abs(got - ref)
    assert np.all(np.isfinite(got)), what
    assert np.linalg.norm(err) / nrm <= rel, f"{what}: rel-L2 {np.linalg.norm(err) / nrm:.3e}"
    assert err.max() <= mx * rms, f"{what}: max-abs {err.max() / rms:.3e} RMS"


@pytest.mark.parametrize("kw,iters", [
    (dict(S=4, B=2, K=16, k0=300, T=72, dtype="ci16", n_pulses=2, blocks=2, kappa=4.0), 25),
    (dict(S=4, B=3, K=488, k0=24, T=200, dtype="ci8", n_pulses=3, blocks=2, kappa=4.5), 25),
    (dict(S=3, B=2, K=24, k0=100, T=40, dtype="ci8", stec=(8.0, 12.0), n_pulses=2, blocks=2, kappa=4.0), 7),
    # even and minimal iteration counts: the x update is applied every other iteration, the last one must not be lost
    (dict(S=3, B=2, K=24, k0=100, T=56, dtype="ci8", n_pulses=2, blocks=2, kappa=4.0), 8),
    (dict(S=3, B=2, K=24, k0=100, T=56, dtype="ci8", n_pulses=2, blocks=2, kappa=4.0), 2),
    (dict(S=3, B=2, K=24, k0=100, T=56, dtype="ci8", n_pulses=2, blocks=2, kappa=4.0), 1),
])
def test_lsmr_inversion_parity(torch, oracle, kw, iters):
    """LOFAR_INV_LSMR against O11 (= scipy's lsmr, pinned): whole chain, two blocks (the 15 carried slices are rows of
    the second block's system), several scratch chunks, sigma and candidates from the LSMR series."""
    w = synth.small(**kw)
    tau, blocks = _blocks(w)
    pipe = oracle.OraclePipeline(tau=tau, stec=np.asarray(w.stec), K=w.K, k0=w.k0, kappa=w.kappa, inversion="lsmr",
                                 lsmr_iters=iters)
    p = binding.plan_for(w, tau)
    p.set_trigger(w.kappa, 1, 1 << 16)
    p.set_inversion(binding.LOFAR_INV_LSMR, iters)
    p.set_scratch_limit(w.B * w.K * 8 * 64)
    offset = 0
    for i, X in enumerate(blocks):
        ref, sig_ref, _, _ = pipe.run_block(X)
        got, rec, n, sigma, _, _ = _run(torch, p, X, w.T)
        for s in range(w.nseries):
            _close(got[s], ref[s], f"block {i} series {s}", LSMR_TOL["rel"], LSMR_TOL["mx"])
        np.testing.assert_allclose(sigma, sig_ref, rtol=2e-5)
        env, sig = oracle_snr(oracle, ref, 1)
        check_candidates(rec, n, env, sig, w.B, w.D, w.kappa, offset)
        offset += w.T * 1024
    # the stage call alone, on caller-owned beam sums
    ns, K, k0, T = 2, 31, 481, 37
    q = binding.Plan(1, K, ns, 16, 0.0)
    q.set_band(k0)
    q.set_input(binding.LOFAR_CI8, T)
    q.set_inversion(binding.LOFAR_INV_LSMR, 12)
    Z = synth.random_z(5, ns, K, T)
    out = torch.empty((ns, T * 1024), dtype=torch.float32, device="cuda")
    q.inverse_ppf(torch.from_numpy(np.ascontiguousarray(Z.view(np.float32).reshape(ns, K, T, 2))).cuda(), T, out)
    torch.cuda.synchronize()
    h = oracle.prototype()
    for s in range(ns):
        y = oracle.idft(Z[s].astype(np.complex128), k0)
        refs = oracle.lsmr_inversion(np.concatenate([np.zeros((15, 1024)), y]), h, 12)
        _close(out[s].cpu().numpy(), refs, f"stage call series {s}", LSMR_TOL["rel"], LSMR_TOL["mx"])
    p.destroy()
    q.destroy()


# ------------------------------------------------------------------------------------------ f2
@pytest.mark.parametrize("kw,lsmr", [
    (dict(S=4, B=2, K=488, k0=24, T=104, dtype="ci8", stec=(12.0,), pulse_stec=12.0, n_pulses=3, blocks=3, kappa=4.5), False),
    (dict(S=3, B=2, K=64, k0=200, T=44, dtype="ci16", stec=(8.0, 10.0, 12.0), pulse_stec=10.0, n_pulses=3, blocks=2, kappa=4.0), False),
    (dict(S=3, B=1, K=100, k0=300, T=32, dtype="ci8", stec=(10.0, 20.0), pulse_stec=10.0, n_pulses=2, blocks=2, kappa=4.0), True),
])
def test_exact_dedispersion_parity(torch, oracle, kw, lsmr):
    """LOFAR_DEDISP_EXACT against O12 (overlap-save rfft * D * irfft per trial on the series reconstructed without
    dispersion phase), whole chain, consecutive blocks (two carried slices of the undispersed series + the PPF
    history), T not a multiple of the 14-slice hop; once combined with the LSMR inversion."""
    w = synth.small(**kw)
    tau, blocks = _blocks(w)
    pipe = oracle.OraclePipeline(tau=tau, stec=np.asarray(w.stec), K=w.K, k0=w.k0, kappa=w.kappa, dedisp="exact",
                                 inversion="lsmr" if lsmr else "matched", lsmr_iters=9)
    p = binding.plan_for(w, tau)
    p.set_trigger(w.kappa, 1, 1 << 16)
    p.set_dedispersion(binding.LOFAR_DEDISP_EXACT)
    if lsmr:
        p.set_inversion(binding.LOFAR_INV_LSMR, 9)
    p.set_scratch_limit(w.B * w.K * 8 * 32)
    tol = LSMR_TOL if lsmr else dict(rel=1e-5, mx=1e-4)
    offset = 0
    state = None
    for i, X in enumerate(blocks):
        ref, sig_ref, _, _ = pipe.run_block(X)
        got, rec, n, sigma, _, _ = _run(torch, p, X, w.T)
        for s in range(w.nseries):
            _close(got[s], ref[s], f"block {i} series {s}", tol["rel"], tol["mx"])
        np.testing.assert_allclose(sigma, sig_ref, rtol=2e-5)
        env, sig = oracle_snr(oracle, ref, 1)
        check_candidates(rec, n, env, sig, w.B, w.D, w.kappa, offset)
        offset += w.T * 1024
        if i == 0:
            state = p.get_state()
            second = got
    # resume from the checkpoint taken after block 0: the two carried slices travel with the state
    q = binding.plan_for(w, tau)
    q.set_trigger(w.kappa, 1, 1 << 16)
    q.set_dedispersion(binding.LOFAR_DEDISP_EXACT)
    if lsmr:
        q.set_inversion(binding.LOFAR_INV_LSMR, 9)
    q.set_state(state)
    got_q, _, _, _, _, _ = _run(torch, q, blocks[1], w.T)
    p.stream_reset()
    _run(torch, p, blocks[0], w.T)
    got_p, _, _, _, _, _ = _run(torch, p, blocks[1], w.T)
    assert np.array_equal(got_q, got_p)
    p.destroy()
    q.destroy()


# ------------------------------------------------------------------------------------------ f4
def test_two_stage_beamforming_parity(torch, oracle):
    """stage 1 forms one pre-beam per sub-array (its stations summed towards the pointing centre),
    lofar_requantize turns those into int16 pseudo-stations, stage 2 runs the whole chain on them.
    Against the oracle doing the same two stages (O4, O13, O4..O8), element by element."""
    w = synth.small(S=6, B=3, K=24, k0=150, T=72, dtype="ci8", stec=(10.0,), n_pulses=2, kappa=4.0)
    tau, blocks = _blocks(w)
    X = blocks[0]
    groups = [(0, 1, 2), (3, 4, 5)]
    scale = 16.0
    tau2 = np.stack([tau[:, list(st)].mean(axis=1) for st in groups], axis=1)          # [B][G]
    # ---- oracle: stage 1 per group (unit weights, no dispersion), re-quantise, stage 2 chain
    X2_ref = np.zeros((len(groups), 2, w.K, w.T, 2), dtype=np.int16)
    W1, D1 = oracle.tables(np.zeros((1, 3)), np.zeros(1), w.K, w.k0)
    for g, st in enumerate(groups):
        Zg = oracle.beamform(np.ascontiguousarray(X[list(st)]), W1, D1)
        X2_ref[g, 0] = oracle.requantise(Zg[0], scale)
    pipe = oracle.OraclePipeline(tau=tau2, stec=np.asarray(w.stec), K=w.K, k0=w.k0, kappa=w.kappa)
    ref, sig_ref, _, _ = pipe.run_block(X2_ref)
    # ---- GPU: one stage-1 plan per group, lofar_requantize into the stage-2 input, stage-2 plan on int16
    X2 = torch.zeros((len(groups), 2, w.K, w.T, 2), dtype=torch.int16, device="cuda")
    for g, st in enumerate(groups):
        p1 = binding.Plan(3, w.K, 1, 16, 0.0)
        p1.set_band(w.k0)
        p1.set_delays(np.zeros((1, 3)))
        p1.set_input(binding.LOFAR_CI8, w.T)
        Z = torch.empty((1, w.K, w.T, 2), dtype=torch.float32, device="cuda")
        p1.beamform_dedisperse(torch.from_numpy(np.ascontiguousarray(X[list(st)])).cuda(), w.T, Z)
        p1.requantize(Z, w.T, scale, X2[g])
        torch.cuda.synchronize()
        p1.destroy()
    assert np.array_equal(X2.cpu().numpy(), X2_ref)                 # integers: bit-exact
    p2 = binding.Plan(len(groups), w.K, w.B, 16, w.stec[0])
    p2.set_band(w.k0)
    p2.set_delays(tau2)
    p2.set_input(binding.LOFAR_CI16, w.T)
    p2.set_trigger(w.kappa, 1, 1 << 16)
    series, cand, count, sigma = binding.new_outputs(p2, w.T)
    p2.run_block(X2, w.T, series, cand, count, sigma)
    torch.cuda.synchronize()
    got = series.cpu().numpy()
    for s in range(w.B):
        assert_close(got[s], ref[s], f"series {s}")
    np.testing.assert_allclose(sigma.cpu().numpy(), sig_ref, rtol=5e-6)
    env, sig = oracle_snr(oracle, ref, 1)
    check_candidates(binding.candidates_to_numpy(cand, count), int(count.item()), env, sig, w.B, 1, w.kappa)
    # ties to even and clipping of the re-quantiser on hand-made values
    z = torch.tensor([[0.5, 1.5], [2.5, -0.5], [1e9, -1e9], [-0.49, 0.51]], dtype=torch.float32, device="cuda")
    q = binding.Plan(1, 1, 1, 16, 0.0)
    q.set_input(binding.LOFAR_CI16, 4)
    out = torch.zeros((1, 2, 1, 4, 2), dtype=torch.int16, device="cuda")
    q.requantize(z.reshape(1, 1, 4, 2), 4, 1.0, out)
    torch.cuda.synchronize()
    assert out[0, 0, 0].cpu().tolist() == [[0, 2], [2, 0], [32767, -32767], [0, 1]] and int(out[0, 1].abs().sum()) == 0
    p2.destroy()
    q.destroy()
