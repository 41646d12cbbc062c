/*
 * lofar_moon.h -- C ABI of the B200-native hot path of the LOFAR lunar-pulse trigger
 * pipeline (arXiv 1612.06592, "Realtime processing of LOFAR data for the detection of
 * nano-second pulses from the Moon").
 *
 * The path (section 2, "Overview of the online data analysis processing
 * steps"): station sub-band voltages -> tied-array beams with the ionospheric
 * de-dispersion phase folded into the per-sub-band weight (re-formulation of
 * BASELINE.json:north_star) -> inversion of the polyphase filter, i.e. inverse Fourier
 * transform + synthesis FIR (the FIR is the matched synthesis H^T, reading A8
 * in DESIGN.md) -> amplitude trigger.
 *
 * Conventions
 *   S stations, 2 polarisations, B beams, D STEC trials, K selected sub-bands k0..k0+K-1 of
 *   an M = 1024 point critically sampled filter bank with P = 16 taps per branch,
 *   T time slices per call.  nseries = B*D; series index = b*D + d.
 *   f_sb(k) = f_zone + k*clock/M.
 *
 * Pointers: unless a parameter name ends in _host, every data pointer is a DEVICE pointer
 * owned by the caller; the library never frees or reallocates caller memory.  The plan owns
 * its tables, the carried PPF history, scratch and the streaming staging buffers.
 * `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Stage
 * calls only enqueue work on `stream` and return without synchronising.
 *
 * Errors: every call returns a lofar_status; nothing aborts or throws across the boundary.
 * There is no CPU fallback: without a CUDA device the calls return LOFAR_E_CUDA.
 * Calls on one plan must be issued from one thread at a time and, because the inverse PPF
 * carries history, in stream order.
 */
#ifndef LOFAR_MOON_H
#define LOFAR_MOON_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(LOFAR_MOON_BUILD)
#define LOFAR_API __attribute__((visibility("default")))
#else
#define LOFAR_API
#endif

typedef struct lofar_plan lofar_plan; /* opaque, owned by the library */

typedef enum {
    LOFAR_OK = 0,
    LOFAR_E_INVALID = 1,  /* NULL pointer, non-positive size, unsupported parameter value      */
    LOFAR_E_SHAPE = 2,    /* sub-band range outside 0..M/2-1, state blob of another plan shape  */
    LOFAR_E_ALIGN = 3,    /* X base or row pitch not 16-byte aligned                           */
    LOFAR_E_ALLOC = 4,    /* host or device allocation failed                                  */
    LOFAR_E_CUDA = 5,     /* a CUDA runtime call failed (sticky error left for the caller)     */
    LOFAR_E_OVERFLOW = 6, /* more candidates than max_candidates (reported by lofar_stream_sync) */
    LOFAR_E_STATE = 7     /* call not legal in the plan's current state, e.g. slices > the
                             max_slices fixed by lofar_plan_set_input          */
} lofar_status;

typedef enum { LOFAR_CI8 = 0, LOFAR_CI16 = 1 } lofar_dtype;

/* One trigger candidate (24 bytes).  With D > 1 trials only the best trial of a
 * (beam, sample) is reported (BASELINE.json:configs[3], reading A15). */
typedef struct {
    uint32_t series; /* b*D + d                                                    */
    uint32_t trial;  /* d                                                          */
    uint64_t sample; /* global 5 ns index = stream offset + q*1024 + r             */
    float env;       /* envelope e[n] (= |xhat[n]| for env_window 1)               */
    float sigma;     /* sigma of that series over this block                       */
} lofar_candidate;

/* One event = a run of candidates of one beam whose samples differ by at most `gap` (48 bytes;
 * reading A22 in DESIGN.md). */
typedef struct {
    uint32_t beam;          /* series / D                                              */
    uint32_t count;         /* candidates merged into the event                        */
    uint64_t first_sample;  /* global 5 ns index of the first and                      */
    uint64_t last_sample;   /* ... the last candidate                                  */
    uint64_t peak_sample;   /* the candidate with the largest env/sigma                */
    uint32_t peak_trial;    /* (lowest sample on exact ties), its trial,               */
    float peak_env;         /* envelope,                                               */
    float peak_sigma;       /* reference level                                         */
    float peak_snr;         /* and env/sigma                                           */
} lofar_event;

typedef enum { LOFAR_SIGMA_BLOCK = 0, LOFAR_SIGMA_CAUSAL = 1 } lofar_sigma_mode;
typedef enum { LOFAR_INV_MATCHED = 0, LOFAR_INV_LSMR = 1 } lofar_inversion;
typedef enum { LOFAR_DEDISP_SUBBAND = 0, LOFAR_DEDISP_EXACT = 1 } lofar_dedispersion;

/* ---- plan ---------------------------------------------------------------------------------
 * BASELINE.json:north_star: "lofar_plan_create(stations, subbands, beams, taps, STEC)".
 * Creates a plan with one trial (D = 1) at stec_tecu, sub-bands k0 = 0..subbands-1 until
 * lofar_plan_set_band moves them, zero delays, the default Kaiser prototype
 * (BASELINE.json:configs[0]: 16384-tap windowed sinc, cutoff 1/1024, beta = 9), int8 input,
 * kappa = 6, env_window = 1, max_candidates = 65536.  taps must be 16 (LOFAR_E_INVALID
 * otherwise).  Device tables are built lazily at the first compute call. */
LOFAR_API lofar_status lofar_plan_create(lofar_plan **out, int stations, int subbands, int beams,
                                         int taps, double stec_tecu);
LOFAR_API void lofar_plan_destroy(lofar_plan *plan);

/* Setters copy their arguments.  Any of them invalidates the device tables;
 * every setter also resets the carried history and the stream offset (as lofar_stream_reset). */
/* first_subband = k0 >= 0, k0 + K <= 512; fft_size must be 1024. */
LOFAR_API lofar_status lofar_plan_set_band(lofar_plan *plan, int first_subband, double f_zone_hz,
                                           double clock_hz, int fft_size);
/* tau_s_host[beams][stations]: arrival lag in seconds of station s for beam b relative to the
 * phase centre (reading A3/A4); weight W[b,s,k] = exp(+2 pi i f_sb(k) tau[b,s]). */
LOFAR_API lofar_status lofar_plan_set_delays(lofar_plan *plan, const double *tau_s_host);
/* D = ntrials >= 1 STEC values in TECU; Dph[d,k] = exp(-2 pi i 1.343e9 STEC_d / f_sb(k)). */
LOFAR_API lofar_status lofar_plan_set_trials(lofar_plan *plan, int ntrials,
                                             const double *stec_tecu_host);
/* h_host[16*1024] analysis prototype (sum = 1); NULL restores the default Kaiser design.
 * The synthesis taps are g = 1024*h (matched synthesis). */
LOFAR_API lofar_status lofar_plan_set_filter(lofar_plan *plan, const double *h_host);
/* Input sample type and the largest `slices` any later call will pass (a larger value returns
 * LOFAR_E_STATE from the compute calls). */
LOFAR_API lofar_status lofar_plan_set_input(lofar_plan *plan, lofar_dtype dtype, int max_slices);
/* Threshold kappa (candidate iff e/sigma > kappa, strict), envelope window W >= 1 samples
 * (e[n] = sqrt(mean of xhat[n-W+1..n]^2), reading A13), candidate buffer capacity. */
LOFAR_API lofar_status lofar_plan_set_trigger(lofar_plan *plan, double kappa, int env_window,
                                              uint32_t max_candidates);
/* How the polyphase filter is inverted after the inverse DFT.  LOFAR_INV_MATCHED (default):
 * one application of the matched synthesis FIR g = 1024 h (= H^T, reading A8; BASELINE.json:north_star).
 * LOFAR_INV_LSMR: the paper's method -- the FIR system H x = y, which decouples into
 * one banded system per residue r (rows: the 15 carried slices and the T slices of the block, unknowns:
 * slices -15 .. T+14, output: slices 0 .. T-1, reading A23), solved by `iterations` (> 0; the paper: ~25)
 * LSMR iterations from x = 0 with no stopping test.  Costs 4 work vectors of (T+30)*4096 bytes per series
 * plus the inverse-DFT rows; needs a series buffer (not trigger-only).  The carried state is the same
 * 15-slice history. */
LOFAR_API lofar_status lofar_plan_set_inversion(lofar_plan *plan, lofar_inversion mode, int iterations);
/* Where the ionospheric dispersion is removed.  LOFAR_DEDISP_SUBBAND (default): one phase per
 * sub-band folded into the beam weight / applied to the beam sums (BASELINE.json:north_star, reading A9).
 * LOFAR_DEDISP_EXACT: the paper's order -- beams are formed and the polyphase filter is
 * inverted WITHOUT dispersion phase (one inversion per beam), then every trial multiplies the spectrum of the
 * 5 ns series by exp(-2 pi i 1.343e9 STEC / f) at the exact frequency of each bin: overlap-save with
 * 16384-sample transforms of which one slice at either end is discarded (reading A24; valid while the
 * dispersive delay across the band stays below one slice, STEC <= 40 TECU for the HBA band).  The output
 * series, sigma and candidate sample indices run ONE SLICE (1024 samples) behind the input: sample n of the
 * output is time n - 1024 of the stream.  Carried state grows by two slices of the undispersed series per
 * beam.  Not available in trigger-only mode; lofar_run_block / lofar_stream_push only (the stage calls keep
 * their definitions). */
LOFAR_API lofar_status lofar_plan_set_dedispersion(lofar_plan *plan, lofar_dedispersion mode);
/* Reference level of the trigger (the recovered signal is used "only
 * to trigger the read-out", so the threshold must be known while a block is reconstructed).
 * LOFAR_SIGMA_BLOCK (default): candidates of a block are measured against the envelope RMS of that
 * block (reading A14).  LOFAR_SIGMA_CAUSAL: block i is measured against sigma of block i-1 of the same
 * series (reading A21); the first block after a reset uses sigma_init_host[B*D] if not NULL, else its own
 * sigma.  With the level known in advance the candidates are decided in the inverse-PPF epilogue and
 * lofar_run_block / lofar_stream_push need not write the series (series == NULL).  `sigma` outputs always
 * receive the RMS of the current block; candidate records carry the level they were measured against.
 * Causal mode needs env_window 1 (LOFAR_E_INVALID otherwise, from the compute calls). */
LOFAR_API lofar_status lofar_plan_set_sigma_mode(lofar_plan *plan, lofar_sigma_mode mode,
                                                 const float *sigma_init_host);
/* Device bytes the plan allocates for the current settings: tables (weights, tensor-core operand
 * images, trial phasors, taps, twiddles), 2 x carried history, envelope tail, beam-sum scratch,
 * trigger partials, and the two streaming staging slots (input block, candidates, count, sigma)
 * that lofar_stream_push adds on first use. */
LOFAR_API lofar_status lofar_plan_workspace_bytes(lofar_plan *plan, size_t *bytes);
/* Device-memory hooks (BASELINE.json:north_star "PyTorch used only for device
 * memory"): every plan-owned DEVICE buffer is obtained with alloc(bytes, ctx) (NULL = failure ->
 * LOFAR_E_ALLOC; at least 256-byte aligned) and returned with free_(ptr, ctx); both NULL restores
 * cudaMalloc/cudaFree.  Buffers already held are released first with the allocator that made
 * them (the plan's own streams are drained; work on caller streams must have completed).  The
 * only memory the plan takes elsewhere is 256 bytes of pinned HOST memory for streaming counts. */
LOFAR_API lofar_status lofar_plan_set_allocator(lofar_plan *plan, void *(*alloc)(size_t, void *),
                                                void (*free_)(void *, void *), void *ctx);
/* Upper bound in bytes for the beam-sum scratch (default 16 GiB -- one chunk for a 0.67 s block of 24 beams x 488 sub-bands; all slots together).  A block longer
 * than the chunk is processed chunk by chunk, history handed over on the device. */
LOFAR_API lofar_status lofar_plan_set_scratch_limit(lofar_plan *plan, size_t bytes);
/* Two-lane block pipeline of lofar_run_block / lofar_stream_push (step a6 applied inside a block: the "CUDA
 * streams" of BASELINE.json:north_star (e)).  mode 0 (default): both kernels of every chunk run back to back on
 * the caller's stream.  mode 1: when the tensor-core beamformer is in use (int8 input, >= 4 beams) and the
 * block is longer than one chunk, the block is cut into chunks of `chunk_slices` (0 = 8192; never more than
 * half the scratch limit), the beamformer of chunk c+1 runs on a low-priority plan-owned stream while the
 * inverse PPF of chunk c runs on a high-priority one, on alternating scratch slots; the inverse PPF is planned
 * for 16 SMs fewer (one wave), which the beamformer uses.  The caller's stream forks into the two lanes and
 * joins them again inside the call, so stream order as seen by the caller is unchanged.  The series are
 * bit-identical to mode 0; sigma differs in its summation order only.  Measured on B200:
 * slower than mode 0 for configs[2] (9.8 - 10.1 vs 9.2 ms per block) because the beamformer needs ~40 SMs' worth of
 * issue slots to reach its HBM rate -- kept as an option, off by default. */
LOFAR_API lofar_status lofar_plan_set_overlap(lofar_plan *plan, int mode, int chunk_slices);
/* How lofar_run_block would cut a block of `slices`: slices per scratch chunk, and the number and
 * length (slices) of the independent time spans one inverse-PPF launch is divided into.  Host only;
 * lets tests aim parity windows at chunk and span boundaries. */
LOFAR_API lofar_status lofar_plan_chunking(lofar_plan *plan, int slices, int64_t *chunk_slices,
                                           int *spans, int *span_slices);
/* The same for chunk number `chunk` (0, 1, ...) of a block of `slices`: its first slice, its length
 * (0 once `chunk` is past the end of the block; the last chunk may be shorter and is then cut into its own
 * spans) and the spans of its inverse-PPF launch.  Host only. */
LOFAR_API lofar_status lofar_plan_chunk_info(lofar_plan *plan, int slices, int chunk, int64_t *first_slice,
                                             int64_t *chunk_slices, int *spans, int *span_slices);

/* ---- stage calls (all pointers device) ------------------------------------------------------
 * X: [S][2][K][slices][re,im] int8 or int16, little endian, time fastest; base and row pitch
 * (slices*2*sizeof(sample)) must be multiples of 16 bytes (LOFAR_E_ALIGN otherwise).
 * Z: [B*D][K][slices] float2.   series: [B*D][slices*1024] float, sample n = q*1024 + r. */

/* a1 + a2:  Z[b*D+d][k][q] = Dph[d,k] * sum_s sum_p W[b,s,k] X[s,p,k,q]. */
LOFAR_API lofar_status lofar_beamform_dedisperse(lofar_plan *plan, const void *X, int slices,
                                                 void *Z, void *stream);
/* f4, two-stage beamforming (sub-arrays pre-beamformed on the first cluster, the
 * final beams formed from those on the second; 16-bit integers on the wire).  Turns the output Z
 * [B*D][K][slices] float2 of lofar_beamform_dedisperse into the input of a second plan whose "stations" are
 * these B*D first-stage beams: X2 [B*D][2][K][slices][re,im] int16, polarisation 0 = clip(rint(Z * scale),
 * +-32767) with ties to even, polarisation 1 = 0.  Device pointers; X2 16-byte aligned. */
LOFAR_API lofar_status lofar_requantize(lofar_plan *plan, const void *Z, int slices, float scale, void *X2,
                                        void *stream);
/* a3 + a4: per series and slice an unnormalised 1024-point Hermitian inverse
 * DFT of the K selected bins (all other bins zero), then
 * xhat[q*1024+r] = 1024 * sum_{t<16} h[r+1024 t] * y[q-t][r].  Reads and then replaces the
 * plan's carried 15-slice history (zeros after lofar_stream_reset). */
LOFAR_API lofar_status lofar_inverse_ppf(lofar_plan *plan, const void *Z, int slices, float *series,
                                         void *stream);
/* a5: envelope, sigma[series] = RMS of the envelope over this block,
 * candidates e > kappa*sigma (best trial per (beam, sample) when D > 1), sorted by
 * (beam, sample).  *count receives the true number of candidates; at most max_candidates
 * records are stored (an unspecified subset, still sorted, when count > max_candidates).
 * Candidate sample indices are stream offset + n; the stream offset advances by
 * slices*1024 per lofar_trigger / lofar_run_block call. */
LOFAR_API lofar_status lofar_trigger(lofar_plan *plan, const float *series, int slices,
                                     lofar_candidate *cand, uint32_t *count, float *sigma,
                                     void *stream);
/* The whole chain on one block: a1..a5 with the beam sums kept in plan scratch.
 * series == NULL selects the trigger-only mode: nothing of the 5 ns series is written
 * to HBM; sigma and the candidate list are the same as with a series (same definitions; values within
 * fp32 rounding).  With LOFAR_SIGMA_BLOCK the chunks whose maximum can reach kappa*sigma are recomputed
 * from X after sigma is known (X must stay valid until the call's work has completed, as always); with
 * LOFAR_SIGMA_CAUSAL candidates come out of the first pass.  Needs env_window 1.  With D > 1 and more
 * raw threshold crossings than max_candidates, *count is that raw number (an overflow), not the number of
 * distinct (beam, sample) candidates. */
LOFAR_API lofar_status lofar_run_block(lofar_plan *plan, const void *X, int slices, float *series,
                                       lofar_candidate *cand, uint32_t *count, float *sigma,
                                       void *stream);

/* f3: groups a candidate list as produced by lofar_trigger / lofar_run_block (device pointers, sorted by
 * (beam, sample), *count valid) into events: consecutive candidates of one beam whose samples differ by at
 * most gap_samples.  *nevents receives the number of events, the first max_events are stored in order. */
LOFAR_API lofar_status lofar_cluster(lofar_plan *plan, const lofar_candidate *cand, const uint32_t *count,
                                     uint64_t gap_samples, lofar_event *events, uint32_t *nevents,
                                     uint32_t max_events, void *stream);

/* ---- streaming driver (a6; BASELINE.json:configs[4]) -------------------------------------------
 * lofar_stream_reset: waits for the plan's own streams and resets the stream offset; the carried
 * history is zeroed on the stream of the next compute call (no device-wide synchronisation).
 * lofar_stream_push: X_host is a HOST buffer (pinned for copy/compute overlap; pageable works
 * but serialises) laid out as X above.  The block is copied into one of two plan-owned device
 * buffers on a copy stream while the previous block computes on a compute stream; then
 * lofar_run_block runs on it; then count, sigma[B*D] and the stored candidates are copied to
 * the *_host buffers (any of which may be NULL).  series is a device buffer (never copied to
 * the host) or NULL (trigger-only, see lofar_run_block).  Returns without waiting.  Host result buffers and X_host must stay untouched
 * until lofar_stream_sync returns.
 * lofar_stream_sync: blocks until all pushed blocks are done; returns LOFAR_E_OVERFLOW if any
 * block since the last sync had more candidates than max_candidates. */
LOFAR_API lofar_status lofar_stream_reset(lofar_plan *plan);
LOFAR_API lofar_status lofar_stream_push(lofar_plan *plan, const void *X_host, int slices,
                                         float *series, lofar_candidate *cand_host,
                                         uint32_t *count_host, float *sigma_host);
LOFAR_API lofar_status lofar_stream_sync(lofar_plan *plan);
/* Checkpoint / resume of the carried state: a small header (stream offset,
 * shape), the 15-slice synthesis history [B*D][15][1024] fp32 and the env_window-1 envelope tail.
 * HOST buffers of lofar_stream_state_bytes bytes.  Both calls block: they drain the plan's own
 * streams and copy synchronously (work the caller enqueued on its own streams must have
 * completed).  set_state on a plan of another shape returns LOFAR_E_SHAPE; before
 * lofar_plan_set_input has fixed the capacity both return LOFAR_E_STATE. */
LOFAR_API lofar_status lofar_stream_state_bytes(lofar_plan *plan, size_t *bytes);
LOFAR_API lofar_status lofar_stream_get_state(lofar_plan *plan, void *state_host, size_t bytes);
LOFAR_API lofar_status lofar_stream_set_state(lofar_plan *plan, const void *state_host, size_t bytes);

/* Per-kernel device timing (measurement aid, PAPER-independent).  With profiling enabled every kernel
 * the plan launches is bracketed by CUDA events on its own stream.  lofar_plan_profile_read waits for
 * the recorded events, ADDS the elapsed milliseconds and launch counts since the previous read to
 * ms_host[LOFAR_PROFILE_SLOTS] / launches_host[LOFAR_PROFILE_SLOTS] (index 0 beamform, 1 inverse PPF, 2 trigger
 * kernels, 3 LSMR solve, 4 exact de-dispersion; a "launch" is one bracketed group) and clears them. */
#define LOFAR_PROFILE_SLOTS 5
LOFAR_API lofar_status lofar_plan_profile(lofar_plan *plan, int enable);
LOFAR_API lofar_status lofar_plan_profile_read(lofar_plan *plan, double *ms_host, uint64_t *launches_host);
/* Number of kernel launches the plan has enqueued so far (for bench accounting). */
LOFAR_API uint64_t lofar_plan_launch_count(const lofar_plan *plan);
LOFAR_API const char *lofar_status_string(lofar_status status);

/* ---- allocation-free entry point -------------------------------------------------------------------
 * The stand-alone trigger of lofar_trigger (step a5: sigma = RMS of |x| over the block per series, candidates
 * |x| / sigma > kappa, sorted by (series, sample); one trial per series, env_window 1) for callers that may not
 * allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  It takes no
 * plan and calls no cudaMalloc / cudaFree or allocating library routine: its scratch (per-chunk sums and maxima,
 * the list of flagged chunks) is a fixed file-scope device array of about 6.1 MiB that every GPU holding the
 * library keeps until the process exits.  Limit: ceil(samples / 16384) * nseries <= LOFAR_STATIC_MAX_CHUNKS
 * (e.g. 24 series of 131072 slices = 196608 chunks); beyond it the call returns LOFAR_E_SHAPE ("shape out of
 * range") and launches nothing.
 * series[nseries][series_pitch] (device, series_pitch >= samples, in floats), cand[max_candidates], count[1],
 * sigma[nseries]: device buffers of the caller; offset = global index of sample 0.  Work is enqueued on `stream`;
 * no synchronisation.  Overflow rule as lofar_trigger (R1): *count is the true total.
 * The array is shared by all calls (all threads, all streams) and keeps the last call's contents; every call clears
 * what must start at zero on its own stream.  Calls that overlap on the GPU race on it: order them (one stream, or
 * events between streams). */
#define LOFAR_STATIC_MAX_CHUNKS 524288
LOFAR_API lofar_status lofar_trigger_static(const float *series, int nseries, int64_t samples, int64_t series_pitch,
                                            double kappa, uint64_t offset, lofar_candidate *cand,
                                            uint32_t max_candidates, uint32_t *count, float *sigma, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* LOFAR_MOON_H */
