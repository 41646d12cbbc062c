"""GPU tests of the boundary's own behaviour: allocator hooks, capacity errors, scratch
chunking, checkpoint/resume of the carried state, lazy reset -- plus the small parity cases the full-size
tests cannot aim at (int8 = -128 on the tensor-core path, env_window > 1 through lofar_run_block and
lofar_stream_push, a non-default prototype)."""
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
    return w, tau, synth.generate_block(w, 0, tau=tau)


def _run(torch, p, X, T):
    series, cand, count, sigma = binding.new_outputs(p, T)
    p.run_block(torch.from_numpy(X).cuda(), T, series, cand, count, sigma)
    torch.cuda.synchronize()
    return series.cpu().numpy(), binding.candidates_to_numpy(cand, count), int(count.item()), sigma.cpu().numpy()


def test_counting_allocator_sees_every_plan_buffer(torch):
    """Every device byte the plan holds comes from the hooks: the sum of the requests equals
    lofar_plan_workspace_bytes (staging included once lofar_stream_push has run) and every pointer is
    returned exactly once."""
    w, tau, X = _case(S=4, B=3, K=24, k0=200, T=48, dtype="ci8", kappa=4.5)
    live, log = {}, []

    def alloc(n):
        ptr = torch.cuda.caching_allocator_alloc(n)
        live[ptr] = n
        log.append(n)
        return ptr

    def free(ptr):
        assert ptr in live, "free of a pointer the plan did not get from the hook"
        del live[ptr]
        torch.cuda.caching_allocator_delete(ptr)

    p = binding.plan_for(w, tau)
    p.set_trigger(w.kappa, 3, 1024)
    p.set_allocator(alloc, free)
    want = p.workspace_bytes()
    ref_plan = binding.plan_for(w, tau)             # same settings on cudaMalloc
    ref_plan.set_trigger(w.kappa, 3, 1024)
    s_ref, _, _, _ = _run(torch, ref_plan, X, w.T)
    s_got, _, _, _ = _run(torch, p, X, w.T)
    assert np.array_equal(s_got, s_ref)
    n_tables = len(log)
    assert n_tables >= 10                            # W, Dph, taps, twiddles, images, 2 x history, tail, scratch, partials, maxima
    Xh = torch.from_numpy(X).pin_memory()
    series = torch.empty((w.nseries, w.T * 1024), dtype=torch.float32, device="cuda")
    p.stream_reset()
    p.stream_push(Xh, w.T, series)
    p.stream_sync()
    assert len(log) == n_tables + 8                  # two staging slots x (input, candidates, count, sigma)
    assert sum(log) == want
    assert np.array_equal(series.cpu().numpy(), s_ref)
    p.destroy()
    ref_plan.destroy()
    assert not live, f"{len(live)} plan buffers were never returned"


def test_torch_caching_allocator_and_failure(torch):
    w, tau, X = _case(S=3, B=2, K=12, k0=40, T=64, dtype="ci8", kappa=4.0)
    p = binding.plan_for(w, tau)
    p.set_torch_allocator()
    before = torch.cuda.memory_allocated()
    s1, _, _, _ = _run(torch, p, X, w.T)
    assert torch.cuda.memory_allocated() - before >= w.B * w.K * w.T * 8 + 2 * w.nseries * 15 * 1024 * 4
    p.set_allocator(None, None)                      # back to cudaMalloc: tables rebuilt, same numbers
    s2, _, _, _ = _run(torch, p, X, w.T)
    assert np.array_equal(s1, s2)
    # an allocator that refuses: LOFAR_E_ALLOC, nothing left half-built, plan still usable afterwards
    p.set_allocator(lambda n: 0, lambda ptr: None)
    series, cand, count, sigma = binding.new_outputs(p, w.T)
    st = p.run_block(torch.from_numpy(X).cuda(), w.T, series, cand, count, sigma, allow=range(8))
    assert st == binding.LOFAR_E_ALLOC
    p.set_allocator(None, None)
    s3, _, _, _ = _run(torch, p, X, w.T)
    assert np.array_equal(s1, s3)
    p.destroy()


def test_capacity_is_a_state_error(torch):
    p = binding.Plan(2, 4, 1, 16, 1.0)
    p.set_input(binding.LOFAR_CI8, 64)
    X = torch.zeros(2 * 2 * 4 * 128 * 2, dtype=torch.int8, device="cuda")
    series, cand, count, sigma = binding.new_outputs(p, 128)
    assert p.run_block(X, 128, series, cand, count, sigma, allow=range(8)) == binding.LOFAR_E_STATE
    assert p.run_block(X, 64, series, cand, count, sigma, allow=range(8)) == binding.LOFAR_OK
    torch.cuda.synchronize()
    p.destroy()


@pytest.mark.parametrize("T,limit_slices", [(200, 64), (136, 32), (96, 96)])
def test_scratch_chunks_hand_over_history(torch, oracle, T, limit_slices):
    """A reduced scratch limit forces lofar_run_block through several time chunks (the path configs[2] takes
    at full size: 195312 slices = two chunks of the 16 GiB default): out0 / step0 offsets, scratch reuse and
    the ping-pong history hand-over between the launches."""
    w, tau, X = _case(S=4, B=5, K=24, k0=200, T=T, dtype="ci8", kappa=4.0, n_pulses=2)
    pipe = oracle.OraclePipeline(tau=tau, stec=np.asarray(w.stec), K=w.K, k0=w.k0, kappa=w.kappa)
    ref, sig_ref, _, _ = pipe.run_block(X)
    p = binding.plan_for(w, tau)
    p.set_scratch_limit(w.B * w.K * 8 * limit_slices)
    zc, nspans, span = p.chunking(T)
    assert zc == limit_slices and span % 16 == 0
    got, rec, n, sigma = _run(torch, p, X, T)
    for s in range(w.nseries):
        assert_close(got[s], ref[s], f"series {s}")
        for c0 in range(zc, T, zc):                  # the slices either side of every chunk boundary
            lo, hi = (c0 - 16) * 1024, min(T, c0 + 16) * 1024
            assert_close(got[s, lo:hi], ref[s, lo:hi], f"series {s} chunk boundary {c0}")
    np.testing.assert_allclose(sigma, sig_ref, rtol=5e-6)
    env, sig = oracle_snr(oracle, ref, 1)
    check_candidates(rec, n, env, sig, w.B, w.D, w.kappa)
    # second block: the history written by the last chunk of block 0 is the one block 1 reads
    X1 = synth.generate_block(w, 1, tau=tau)
    ref1, _, _, _ = pipe.run_block(X1)
    got1, _, _, _ = _run(torch, p, X1, T)
    for s in range(w.nseries):
        assert_close(got1[s], ref1[s], f"block 1 series {s}")
    p.destroy()


@pytest.mark.parametrize("T,chunk", [(200, 64), (264, 32)])
def test_two_lane_pipeline_matches_oracle(torch, oracle, T, chunk):
    """lofar_plan_set_overlap(1): the beamformer of chunk c + 1 on one plan stream beside the inverse PPF of chunk c
    on another, alternating scratch slots, fork / join with the caller's stream. Same results as the oracle, and
    bit-identical series to the serial mode; two blocks, so that the slot and history hand-over across the join is
    covered as well."""
    w, tau, X = _case(S=4, B=5, K=24, k0=200, T=T, dtype="ci8", kappa=4.0, n_pulses=2)
    pipe = oracle.OraclePipeline(tau=tau, stec=np.asarray(w.stec), K=w.K, k0=w.k0, kappa=w.kappa)
    ref, sig_ref, _, _ = pipe.run_block(X)
    X1 = synth.generate_block(w, 1, tau=tau)
    ref1, sig1, _, _ = pipe.run_block(X1)
    p = binding.plan_for(w, tau)
    p.set_overlap(1, chunk)
    chunks = p.chunks(T)
    assert len(chunks) == -(-T // chunk) and all(c[1] <= chunk for c in chunks) and sum(c[1] for c in chunks) == T
    q = binding.plan_for(w, tau)                     # serial twin
    q.set_scratch_limit(w.B * w.K * 8 * chunk)
    for blk, (Xb, rb, sb) in enumerate(((X, ref, sig_ref), (X1, ref1, sig1))):
        got, rec, n, sigma = _run(torch, p, Xb, T)
        ser, _, _, sig_serial = _run(torch, q, Xb, T)
        assert np.array_equal(got, ser)
        np.testing.assert_allclose(sigma, sig_serial, rtol=1e-6)
        for s in range(w.nseries):
            assert_close(got[s], rb[s], f"series {s}")
        np.testing.assert_allclose(sigma, sb, rtol=5e-6)
        env, sig = oracle_snr(oracle, rb, 1)
        check_candidates(rec, n, env, sig, w.B, w.D, w.kappa, offset=blk * T * 1024)
    p.destroy()
    q.destroy()


def test_int8_minimum_on_the_tensor_core_path(torch, oracle):
    """-128 is legal int8 input; the tcgen05 kernel (B >= 4) converts bytes to fp16 through an
    offset trick that must stay exact at the end of the range, also for -128 + -128 = -256."""
    w, tau, X = _case(S=24, B=24, K=12, k0=100, T=264, dtype="ci8")
    rng = np.random.default_rng(7)
    X = X.copy()
    X[rng.random(X.shape) < 0.15] = -128
    X[:, :, 3, 40:48, :] = -128                      # both polarisations, all stations: sums of -256
    X[:, :, 5, 100:108, :] = 127
    W, Dph = oracle.tables(tau, np.asarray(w.stec), w.K, w.k0)
    Zref = oracle.beamform(X, W, Dph)
    p = binding.plan_for(w, tau)
    Z = torch.empty((w.nseries, w.K, w.T, 2), dtype=torch.float32, device="cuda")
    p.beamform_dedisperse(torch.from_numpy(X).cuda(), w.T, Z)
    torch.cuda.synchronize()
    Zg = Z.cpu().numpy().view(np.complex64)[..., 0]
    assert_close(Zg.real, Zref.real, "Re Z")
    assert_close(Zg.imag, Zref.imag, "Im Z")
    pipe = oracle.OraclePipeline(tau=tau, stec=np.asarray(w.stec), K=w.K, k0=w.k0, kappa=w.kappa)
    ref, _, _, _ = pipe.run_block(X)
    got, _, _, _ = _run(torch, p, X, w.T)
    for s in range(0, w.nseries, 5):
        assert_close(got[s], ref[s], f"series {s}")
    p.destroy()


@pytest.mark.parametrize("Wn", [8, 3])
def test_env_window_through_run_block_and_stream_push(torch, oracle, Wn):
    """env_window > 1 through the fused calls: the reduce kernel recomputes sigma from the series and the
    W-1 sample tail is carried from block to block."""
    w = synth.small(S=4, B=3, K=24, k0=200, T=48, dtype="ci8", n_pulses=4, blocks=3, kappa=2.2)
    _, _, tau = synth.geometry(w)
    blocks = [synth.generate_block(w, b, tau=tau) for b in range(w.blocks)]
    pipe = oracle.OraclePipeline(tau=tau, stec=np.asarray(w.stec), K=w.K, k0=w.k0, kappa=w.kappa, Wn=Wn)
    p = binding.plan_for(w, tau)
    p.set_trigger(w.kappa, Wn, 1 << 16)
    q = binding.plan_for(w, tau)
    q.set_trigger(w.kappa, Wn, 1 << 16)
    q.stream_reset()
    offset = 0
    tails = [np.zeros(Wn - 1) for _ in range(w.nseries)]
    for X in blocks:
        ref, sig_ref, _, _ = pipe.run_block(X)
        got, rec, n, sigma = _run(torch, p, X, w.T)
        for s in range(w.nseries):
            assert_close(got[s], ref[s], f"series {s}")
        np.testing.assert_allclose(sigma, sig_ref, rtol=5e-6)
        env, sig = oracle_snr(oracle, ref, Wn, tails)
        ndef, _ = check_candidates(rec, n, env, sig, w.B, w.D, w.kappa, offset)
        assert ndef > 0
        # the same block through the streaming driver
        series = torch.empty((w.nseries, w.T * 1024), dtype=torch.float32, device="cuda")
        cand_h = torch.zeros((1 << 16, 24), dtype=torch.uint8).pin_memory()
        count_h = torch.zeros(1, dtype=torch.int32).pin_memory()
        sigma_h = torch.zeros(w.nseries, dtype=torch.float32).pin_memory()
        q.stream_push(torch.from_numpy(X).pin_memory(), w.T, series, cand_h, count_h, sigma_h)
        q.stream_sync()
        assert np.array_equal(series.cpu().numpy(), got)
        rec_s = binding.candidates_to_numpy(cand_h.numpy(), int(count_h.item()))
        assert np.array_equal(rec_s, rec)
        tails = [ref[s, ref.shape[1] - (Wn - 1):] for s in range(w.nseries)]
        offset += w.T * 1024
    p.destroy()
    q.destroy()


def test_non_default_prototype(torch, oracle):
    """lofar_plan_set_filter with a prototype other than the Kaiser default: a Hann-windowed sinc."""
    w, tau, X = _case(S=3, B=2, K=40, k0=100, T=80, dtype="ci16", kappa=4.0)
    n = np.arange(16 * 1024)
    h = np.sinc((n - 8191.5) / 1024.0) * np.hanning(16 * 1024)
    h /= h.sum()
    assert np.max(np.abs(h - oracle.prototype())) > 1e-5
    pipe = oracle.OraclePipeline(tau=tau, stec=np.asarray(w.stec), K=w.K, k0=w.k0, kappa=w.kappa, h=h)
    ref, sig_ref, _, _ = pipe.run_block(X)
    p = binding.plan_for(w, tau)
    p.set_filter(h)
    got, rec, ncand, sigma = _run(torch, p, X, w.T)
    for s in range(w.nseries):
        assert_close(got[s], ref[s], f"series {s}")
    np.testing.assert_allclose(sigma, sig_ref, rtol=5e-6)
    p.set_filter(None)                                # back to the default: differs from the Hann result
    got2, _, _, _ = _run(torch, p, X, w.T)
    assert np.max(np.abs(got2 - got)) > 1e-3 * np.abs(got).max()
    p.destroy()


def test_checkpoint_resume_and_lazy_reset(torch, oracle):
    """lofar_stream_get_state after block 0 + lofar_stream_set_state on a fresh plan = the same block 1,
    bit for bit (history, envelope tail, stream offset); lofar_stream_reset restores the stream start."""
    w = synth.small(S=4, B=3, K=24, k0=200, T=48, dtype="ci8", n_pulses=3, blocks=2, kappa=3.0)
    _, _, tau = synth.geometry(w)
    X0, X1 = (synth.generate_block(w, b, tau=tau) for b in range(2))
    Wn = 4
    a = binding.plan_for(w, tau)
    a.set_trigger(w.kappa, Wn, 1 << 16)
    s0, rec0, n0, sig0 = _run(torch, a, X0, w.T)
    state = a.get_state()
    s1, rec1, n1, sig1 = _run(torch, a, X1, w.T)
    b = binding.plan_for(w, tau)
    b.set_trigger(w.kappa, Wn, 1 << 16)
    b.set_state(state)
    t1, rec1b, n1b, sig1b = _run(torch, b, X1, w.T)
    assert np.array_equal(s1, t1) and n1 == n1b and np.array_equal(rec1, rec1b) and np.array_equal(sig1, sig1b)
    assert rec1.size and rec1["sample"].min() >= w.T * 1024          # offset restored
    # a blob of another shape is refused
    c = binding.Plan(w.S, w.K, w.B + 1, 16, 10.0)
    c.set_input(binding.LOFAR_CI8, w.T)
    assert c.set_state(state, allow=range(8)) == binding.LOFAR_E_SHAPE
    c.destroy()
    # reset: the next call starts the stream again (zero history, offset 0), enqueued on that call's stream
    b.stream_reset()
    r0, recr, nr, sigr = _run(torch, b, X0, w.T)
    assert np.array_equal(r0, s0) and np.array_equal(recr, rec0)
    pipe = oracle.OraclePipeline(tau=tau, stec=np.asarray(w.stec), K=w.K, k0=w.k0, kappa=w.kappa, Wn=Wn)
    ref0, _, _, _ = pipe.run_block(X0)
    ref1, _, _, _ = pipe.run_block(X1)
    for s in range(w.nseries):
        assert_close(s0[s], ref0[s], f"block 0 series {s}")
        assert_close(s1[s], ref1[s], f"block 1 series {s}")
    a.destroy()
    b.destroy()


@pytest.mark.parametrize("trials", [1, 3])
def test_run_block_is_bit_reproducible(torch, trials):
    """compute-sanitizer's racecheck is closed on this GPU pool, so this is the stand-in: the same block three times
    from the same state must give bit-identical series, sigma and candidates. The inverse PPF synchronises its phases
    with split mbarriers (warps run into the next phase), so a missing wait would show up as run-to-run differences;
    the case has 488 sub-bands, many spans per launch and enough steps per span for warps to drift apart."""
    stec = (12.0,) if trials == 1 else (9.0, 12.0, 15.0)
    w, tau, X = _case(S=6, B=8, K=488, k0=24, T=3000, dtype="ci8", stec=stec, n_pulses=3, kappa=5.0)
    p = binding.plan_for(w, tau)
    Xd = torch.from_numpy(X).cuda()
    ref = None
    for _ in range(3):
        p.stream_reset()
        series, cand, count, sigma = binding.new_outputs(p, w.T)
        p.run_block(Xd, w.T, series, cand, count, sigma)
        torch.cuda.synchronize()
        got = (series, sigma.clone(), int(count.item()), cand.clone())
        if ref is None:
            ref = got
            assert torch.isfinite(series).all() and float(series.abs().max()) > 0
        else:
            assert torch.equal(got[0], ref[0]), "series differ between identical runs"
            assert torch.equal(got[1], ref[1]) and got[2] == ref[2]
            assert torch.equal(got[3][:got[2]], ref[3][:ref[2]])
    p.destroy()
