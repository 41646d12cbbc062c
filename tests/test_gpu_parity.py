"""GPU parity tests (pytest -m gpu): the CUDA path, called through the C ABI, against the CPU oracle on
the same seeded inputs.  Tolerances are those of BASELINE.json:north_star (tests/parity_util.py)."""
import numpy as np
import pytest

from paper_1612_06592_b200 import binding, synth
from parity_util import assert_close, check_candidates, oracle_snr

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch():
    import torch as t
    assert t.cuda.is_available(), "GPU tests need a CUDA device"
    binding.load()
    return t


def _case(**kw):
    w = synth.small(**kw)
    _, _, tau = synth.geometry(w)
    X = synth.generate_block(w, 0, tau=tau)
    return w, tau, X


def _pipeline(oracle, w, tau, **kw):
    return oracle.OraclePipeline(tau=tau, stec=np.asarray(w.stec), K=w.K, k0=w.k0, kappa=w.kappa, **kw)


def _cand_np(cand, count):
    return binding.candidates_to_numpy(cand, count)


BEAMFORM_CASES = [
    dict(S=3, B=1, K=12, k0=40, T=64, dtype="ci8"),
    dict(S=4, B=2, K=16, k0=300, T=200, dtype="ci16"),
    dict(S=5, B=3, K=7, k0=1, T=1000, dtype="ci8"),           # K not a multiple of 4, ragged T
    dict(S=24, B=24, K=20, k0=490, T=520, dtype="ci8"),        # full beam count, band touching bin 511
    dict(S=24, B=8, K=9, k0=0, T=264, dtype="ci16", stec=(5.0, 6.0, 7.5)),   # k0 = 0, D = 3
    dict(S=2, B=12, K=5, k0=254, T=72, dtype="ci8"),
    dict(S=7, B=30, K=3, k0=100, T=136, dtype="ci16"),         # more than one beam group
    dict(S=6, B=5, K=4, k0=17, T=8, dtype="ci8"),              # shorter than one step
]


@pytest.mark.parametrize("kw", BEAMFORM_CASES)
def test_beamform_dedisperse_parity(torch, oracle, kw):
    w, tau, X = _case(**kw)
    W, Dph = oracle.tables(tau, np.asarray(w.stec), w.K, w.k0)
    Zref = oracle.beamform(X, W, Dph)
    p = binding.plan_for(w, tau)
    Xd = torch.from_numpy(X).cuda()
    Z = torch.empty((w.nseries, w.K, w.T, 2), dtype=torch.float32, device="cuda")
    p.beamform_dedisperse(Xd, w.T, Z)
    torch.cuda.synchronize()
    Zg = Z.cpu().numpy().view(np.complex64)[..., 0]
    assert_close(Zg.real, Zref.real, "Re Z")
    assert_close(Zg.imag, Zref.imag, "Im Z")
    p.destroy()


IPPF_CASES = [
    dict(nseries=1, K=16, k0=300, T=64),
    dict(nseries=2, K=488, k0=24, T=200),
    dict(nseries=3, K=244, k0=256, T=1000),
    dict(nseries=2, K=512, k0=0, T=48),       # every bin including 0 and 256
    dict(nseries=1, K=3, k0=255, T=33),       # odd T (no 16-byte loads), band around bin 256
    dict(nseries=2, K=31, k0=481, T=5),       # shorter than the history
]


@pytest.mark.parametrize("kw", IPPF_CASES)
def test_inverse_ppf_parity_and_history(torch, oracle, kw):
    ns, K, k0, T = kw["nseries"], kw["K"], kw["k0"], kw["T"]
    h = oracle.prototype()
    p = binding.Plan(1, K, ns, 16, 0.0)     # nseries = B beams, one trial
    p.set_band(k0)
    p.set_input(binding.LOFAR_CI8, T)
    hist = np.zeros((ns, 15, 1024))
    for block in range(3):                  # three consecutive blocks: history carried twice
        Z = synth.random_z(10 * block + T, ns, K, T)
        Zd = torch.from_numpy(np.ascontiguousarray(Z.view(np.float32).reshape(ns, K, T, 2))).cuda()
        out = torch.empty((ns, T * 1024), dtype=torch.float32, device="cuda")
        p.inverse_ppf(Zd, T, out)
        torch.cuda.synchronize()
        got = out.cpu().numpy()
        for s in range(ns):
            y = oracle.idft(Z[s].astype(np.complex128), k0)
            ylead = np.concatenate([hist[s], y], axis=0)
            ref = oracle.synthesis(ylead, h)
            hist[s] = ylead[-15:]
            assert_close(got[s], ref, f"series {s} block {block}")
    p.destroy()


@pytest.mark.parametrize("D,Wn,N", [(1, 1, 40 * 1024), (4, 1, 33 * 1024), (1, 8, 20 * 1024), (3, 5, 17 * 1024)])
def test_trigger_parity(torch, oracle, D, Wn, N):
    B = 3
    ns = B * D
    kappa = 5.0 if Wn == 1 else 2.5      # a one-sample spike of 9 sigma is 9/sqrt(W) in the envelope
    p = binding.Plan(2, 8, B, 16, 5.0)
    if D > 1:
        p.set_trials(np.arange(5.0, 5.0 + D))
    p.set_input(binding.LOFAR_CI8, N // 1024)
    p.set_trigger(kappa, Wn, 4096)
    tails = [np.zeros(Wn - 1) for _ in range(ns)]
    offset = 0
    for block in range(2):
        x = synth.random_series(100 * D + 10 * Wn + block, ns, N)
        xd = torch.from_numpy(x).cuda()
        cand = torch.zeros((4096, 24), dtype=torch.uint8, device="cuda")
        count = torch.zeros(1, dtype=torch.int32, device="cuda")
        sigma = torch.zeros(ns, dtype=torch.float32, device="cuda")
        p.trigger(xd, N // 1024, cand, count, sigma)
        torch.cuda.synchronize()
        env, sig = oracle_snr(oracle, x.astype(np.float64), Wn, tails)
        np.testing.assert_allclose(sigma.cpu().numpy(), sig, rtol=2e-6)
        rec = _cand_np(cand, count)
        ndef, ngot = check_candidates(rec, int(count.item()), env, sig, B, D, kappa, offset)
        assert ndef > 0
        tails = [x[s, N - (Wn - 1):].astype(np.float64) if Wn > 1 else np.zeros(0) for s in range(ns)]
        offset += N
    p.destroy()


RUN_CASES = [
    dict(S=3, B=2, K=12, k0=40, T=64, dtype="ci8", kappa=4.0),
    dict(S=4, B=2, K=16, k0=300, T=200, dtype="ci16", kappa=4.0),
    dict(S=24, B=24, K=40, k0=100, T=104, dtype="ci8", kappa=4.0),
    dict(S=6, B=3, K=33, k0=470, T=72, dtype="ci8", stec=(8.0, 10.0, 12.0, 14.0), kappa=4.0),
]


@pytest.mark.parametrize("kw", RUN_CASES)
def test_run_block_parity(torch, oracle, kw):
    w, tau, X = _case(**kw)
    pipe = _pipeline(oracle, w, tau)
    ref, sig_ref, _, _ = pipe.run_block(X)
    p = binding.plan_for(w, tau)
    p.set_trigger(w.kappa, 1, 1 << 16)
    series, cand, count, sigma = binding.new_outputs(p, w.T)
    p.run_block(torch.from_numpy(X).cuda(), w.T, series, cand, count, sigma)
    torch.cuda.synchronize()
    got = series.cpu().numpy()
    for s in range(w.nseries):
        assert_close(got[s], ref[s], f"series {s}")
    np.testing.assert_allclose(sigma.cpu().numpy(), sig_ref, rtol=5e-6)
    env, sig = oracle_snr(oracle, ref, 1)
    check_candidates(_cand_np(cand, count), int(count.item()), env, sig, w.B, w.D, w.kappa)
    p.destroy()


def test_streaming_matches_oracle_and_one_shot(torch, oracle):
    """configs[4] in miniature: 4 blocks from pinned host memory, pulses at block edges (P9)."""
    w = synth.small(S=4, B=3, K=24, k0=200, T=48, dtype="ci8", n_pulses=6, blocks=4, kappa=4.5)
    _, _, tau = synth.geometry(w)
    blocks = [synth.generate_block(w, b, tau=tau) for b in range(w.blocks)]
    pipe = _pipeline(oracle, w, tau)
    p = binding.plan_for(w, tau)
    p.set_trigger(w.kappa, 1, 8192)
    p.stream_reset()
    outs = []
    for X in blocks:
        Xh = torch.from_numpy(X).pin_memory()
        series = torch.empty((w.nseries, w.T * 1024), dtype=torch.float32, device="cuda")
        cand_h = torch.zeros((8192, 24), dtype=torch.uint8).pin_memory()
        count_h = torch.zeros(1, dtype=torch.int32).pin_memory()
        sigma_h = torch.zeros(w.nseries, dtype=torch.float32).pin_memory()
        p.stream_push(Xh, w.T, series, cand_h, count_h, sigma_h)
        outs.append((Xh, series, cand_h, count_h, sigma_h))
    p.stream_sync()
    offset = 0
    for X, (_, series, cand_h, count_h, sigma_h) in zip(blocks, outs):
        ref, sig_ref, _, _ = pipe.run_block(X)
        got = series.cpu().numpy()
        for s in range(w.nseries):
            assert_close(got[s], ref[s], f"series {s}")
        np.testing.assert_allclose(sigma_h.numpy(), sig_ref, rtol=5e-6)
        env, sig = oracle_snr(oracle, ref, 1)
        rec = binding.candidates_to_numpy(cand_h.numpy(), int(count_h.item()))
        check_candidates(rec, int(count_h.item()), env, sig, w.B, w.D, w.kappa, offset)
        offset += w.T * 1024
    # one-shot on the concatenation gives the same series (sigma is per block by definition)
    Xall = np.ascontiguousarray(np.concatenate(blocks, axis=3))
    p2 = binding.plan_for(synth.small(S=4, B=3, K=24, k0=200, T=48 * 4, dtype="ci8", kappa=4.5), tau)
    series, cand, count, sigma = binding.new_outputs(p2, 48 * 4)
    p2.run_block(torch.from_numpy(Xall).cuda(), 48 * 4, series, cand, count, sigma)
    torch.cuda.synchronize()
    one = series.cpu().numpy()
    cat = np.concatenate([o[1].cpu().numpy() for o in outs], axis=1)
    assert np.max(np.abs(one - cat)) <= 1e-6 * np.sqrt(np.mean(one.astype(np.float64) ** 2)) * 10
    p.destroy()
    p2.destroy()


def test_error_paths(torch):
    p = binding.Plan(2, 4, 1, 16, 1.0)
    p.set_input(binding.LOFAR_CI8, 64)
    X = torch.zeros(2 * 2 * 4 * 64 * 2 + 64, dtype=torch.int8, device="cuda")
    Z = torch.empty((1, 4, 64, 2), dtype=torch.float32, device="cuda")
    assert p.beamform_dedisperse(X, 0, Z, allow=range(8)) == binding.LOFAR_E_INVALID
    assert p.beamform_dedisperse(X, 128, Z, allow=range(8)) == binding.LOFAR_E_STATE      # beyond max_slices
    assert p.beamform_dedisperse(X[1:], 64, Z, allow=range(8)) == binding.LOFAR_E_ALIGN
    assert p.beamform_dedisperse(X, 4, Z, allow=range(8)) == binding.LOFAR_E_ALIGN      # 8-byte row pitch
    assert p.beamform_dedisperse(X, 64, None, allow=range(8)) == binding.LOFAR_E_INVALID
    assert p.beamform_dedisperse(X, 64, Z, allow=range(8)) == binding.LOFAR_OK
    torch.cuda.synchronize()
    p.destroy()


def test_candidate_overflow_reports_true_count(torch):
    w, tau, X = _case(S=3, B=2, K=12, k0=40, T=64, dtype="ci8", kappa=1.0)
    p = binding.plan_for(w, tau)
    p.set_trigger(1.0, 1, 128)
    series, cand, count, sigma = binding.new_outputs(p, w.T)
    p.run_block(torch.from_numpy(X).cuda(), w.T, series, cand, count, sigma)
    torch.cuda.synchronize()
    x = series.cpu().numpy().astype(np.float64)
    sig = sigma.cpu().numpy().astype(np.float64)
    expect = int((np.abs(x) > 1.0 * sig[:, None]).sum())
    assert abs(int(count.item()) - expect) <= max(8, expect // 2000)    # fp32 vs fp64 at the threshold
    assert int(count.item()) > 128
    rec = binding.candidates_to_numpy(cand, 128)
    key = (rec["series"].astype(np.int64) << 40) + rec["sample"].astype(np.int64)
    assert np.all(np.diff(key) > 0)
    p.destroy()
