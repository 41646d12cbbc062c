// api.cu -- the C ABI (include/lofar_moon.h): plan, host-side double-precision tables, workspace,
// the stage calls, the fused block call and the double-buffered streaming driver (step a6).
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>

#include "plan.h"

using namespace lofar;

namespace {

constexpr double kTwoPi = 6.283185307179586476925286766559;
constexpr double kDispersion = 1.343e9;   // phi(f) = 2 pi * 1.343e9 * STEC / f  (BASELINE.json:configs[0])
constexpr int kMfft = 1024, kTaps = 16, kHalf = 512, kStepSlices = 16;
constexpr size_t kScratchBudget = (size_t)4 << 30;   // bytes of beam-sum scratch per time chunk
constexpr int kCountRing = 64;

#define CU(call)                                   \
    do {                                           \
        if ((call) != cudaSuccess) return LOFAR_E_CUDA; \
    } while (0)

template <typename T>
lofar_status dev_alloc(lofar_plan *p, T **ptr, size_t count)
{
    *ptr = nullptr;
    if (count == 0) return LOFAR_OK;
    void *v = nullptr;
    cudaError_t e = cudaMalloc(&v, count * sizeof(T));
    if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); return LOFAR_E_ALLOC; }
    if (e != cudaSuccess) return LOFAR_E_CUDA;
    *ptr = static_cast<T *>(v);
    p->device_bytes += count * sizeof(T);
    return LOFAR_OK;
}

template <typename T>
void dev_free(T *&ptr)
{
    if (ptr) cudaFree(ptr);
    ptr = nullptr;
}

void free_tables(lofar_plan *p)
{
    dev_free(p->dWimg);
    dev_free(p->dW); dev_free(p->dDph); dev_free(p->dGs); dev_free(p->dTw);
    dev_free(p->dHist[0]); dev_free(p->dHist[1]); dev_free(p->dTail);
    dev_free(p->dZ); dev_free(p->dPartial); dev_free(p->dChunkMax);
    for (int i = 0; i < 2; ++i) { dev_free(p->dX[i]); dev_free(p->dCand[i]); dev_free(p->dCount[i]); dev_free(p->dSigma[i]); }
    p->dX_bytes = 0;
    p->device_bytes = 0;
    p->built = false;
}

// Default prototype: Kaiser-windowed sinc, cutoff 1/1024 of Nyquist, beta = 9, unit DC gain
// (BASELINE.json:configs[0]; reading A7).
void default_prototype(std::vector<double> &h)
{
    const int L = kMfft * kTaps;
    h.resize(L);
    const double beta = 9.0, centre = 0.5 * (L - 1);
    const double denom = std::cyl_bessel_i(0.0, beta);
    double total = 0.0;
    for (int n = 0; n < L; ++n) {
        const double x = (n - centre) / kMfft;
        const double sinc = (x == 0.0) ? 1.0 : std::sin(M_PI * x) / (M_PI * x);
        const double u = (n - centre) / centre;
        const double win = std::cyl_bessel_i(0.0, beta * std::sqrt(std::fmax(0.0, 1.0 - u * u))) / denom;
        h[n] = sinc * win;
        total += h[n];
    }
    for (int n = 0; n < L; ++n) h[n] /= total;
}

float2 unit_phasor(double turns)
{
    turns -= std::floor(turns);
    return make_float2((float)std::cos(kTwoPi * turns), (float)std::sin(kTwoPi * turns));
}

// Brackets the kernels launched inside its lifetime with two events on their stream.
struct ProfScope {
    lofar_plan *p; int id; cudaStream_t st; cudaEvent_t a = nullptr, b = nullptr;
    static cudaEvent_t take(lofar_plan *p)
    {
        cudaEvent_t e = nullptr;
        if (!p->prof_pool.empty()) { e = p->prof_pool.back(); p->prof_pool.pop_back(); }
        else cudaEventCreate(&e);
        return e;
    }
    ProfScope(lofar_plan *p_, int id_, cudaStream_t st_) : p(p_), id(id_), st(st_)
    {
        if (p->prof) { a = take(p); b = take(p); cudaEventRecord(a, st); }
    }
    ~ProfScope()
    {
        if (a) { cudaEventRecord(b, st); p->prof_pending.push_back({id, a, b}); }
    }
};

long long round_up(long long v, long long m) { return (v + m - 1) / m * m; }

size_t sample_bytes(const lofar_plan *p) { return p->dtype == LOFAR_CI16 ? 4 : 2; }

lofar_status build(lofar_plan *p)
{
    free_tables(p);
    int dev = 0;
    CU(cudaGetDevice(&dev));
    CU(cudaDeviceGetAttribute(&p->num_sms, cudaDevAttrMultiProcessorCount, dev));
    if (ippf_configure() != 0) return LOFAR_E_CUDA;
    const int S = p->S, K = p->K, B = p->B, D = p->D, ns = B * D;

    // ---- tables, in double on the host, rounded once to fp32 ----
    std::vector<float2> W((size_t)K * B * S), Dph((size_t)D * K), gs((size_t)kTaps * kHalf), tw(256 + 512);
    const bool tc = p->dtype == LOFAR_CI8 && S <= 32 && B <= 128;
    const size_t img = tc ? tc_image_halfs(S, B) : 0;
    std::vector<unsigned short> wimg((size_t)K * 2 * img);
    std::vector<double> wre((size_t)B * S), wim((size_t)B * S);
    for (int j = 0; j < K; ++j) {
        const double f = p->f_zone + (double)(p->k0 + j) * (p->clock / kMfft);
        for (int d = 0; d < D; ++d) Dph[(size_t)d * K + j] = unit_phasor(-(kDispersion * p->stec[d] / f));
        const double fold = (D == 1) ? -(kDispersion * p->stec[0] / f) : 0.0;   // one trial: fold the phase into W
        for (int b = 0; b < B; ++b)
            for (int s = 0; s < S; ++s) {
                double turns = f * p->tau[(size_t)b * S + s] + (fold - std::floor(fold));
                turns -= std::floor(turns);
                W[((size_t)j * B + b) * S + s] = unit_phasor(turns);
                wre[(size_t)b * S + s] = std::cos(kTwoPi * turns);
                wim[(size_t)b * S + s] = std::sin(kTwoPi * turns);
            }
        if (tc) tc_build_image(wre.data(), wim.data(), S, B, &wimg[(size_t)j * 2 * img], &wimg[((size_t)j * 2 + 1) * img]);
    }
    for (int t = 0; t < kTaps; ++t)
        for (int n = 0; n < kHalf; ++n)
            gs[(size_t)t * kHalf + n] = make_float2((float)(kMfft * p->h[2 * n + kMfft * t]),
                                                    (float)(kMfft * p->h[2 * n + 1 + kMfft * t]));
    // twiddles: w1024[256] for the pre-pass, TB[r][j] = exp(2 pi i j r / 512) (r < 32, j < 16) for the radix-32 pass
    for (int m = 0; m < 256; ++m) tw[m] = unit_phasor((double)m / 1024.0);
    for (int r = 0; r < 32; ++r)
        for (int jj = 0; jj < 16; ++jj) tw[256 + r * 16 + jj] = unit_phasor((double)(jj * r) / 512.0);

    lofar_status st;
    if ((st = dev_alloc(p, &p->dW, W.size())) != LOFAR_OK) return st;
    if ((st = dev_alloc(p, &p->dDph, Dph.size())) != LOFAR_OK) return st;
    if ((st = dev_alloc(p, &p->dGs, gs.size())) != LOFAR_OK) return st;
    if ((st = dev_alloc(p, &p->dTw, tw.size())) != LOFAR_OK) return st;
    if (tc) {
        if ((st = dev_alloc(p, &p->dWimg, wimg.size())) != LOFAR_OK) return st;
        CU(cudaMemcpy(p->dWimg, wimg.data(), wimg.size() * sizeof(unsigned short), cudaMemcpyHostToDevice));
    }
    CU(cudaMemcpy(p->dW, W.data(), W.size() * sizeof(float2), cudaMemcpyHostToDevice));
    CU(cudaMemcpy(p->dDph, Dph.data(), Dph.size() * sizeof(float2), cudaMemcpyHostToDevice));
    CU(cudaMemcpy(p->dGs, gs.data(), gs.size() * sizeof(float2), cudaMemcpyHostToDevice));
    CU(cudaMemcpy(p->dTw, tw.data(), tw.size() * sizeof(float2), cudaMemcpyHostToDevice));

    // ---- carried state ----
    const size_t hist = (size_t)ns * (kTaps - 1) * kMfft;
    for (int i = 0; i < 2; ++i) {
        if ((st = dev_alloc(p, &p->dHist[i], hist)) != LOFAR_OK) return st;
        CU(cudaMemset(p->dHist[i], 0, hist * sizeof(float)));
    }
    p->hist_parity = 0;
    if (p->env_window > 1) {
        if ((st = dev_alloc(p, &p->dTail, (size_t)ns * (p->env_window - 1))) != LOFAR_OK) return st;
        CU(cudaMemset(p->dTail, 0, (size_t)ns * (p->env_window - 1) * sizeof(float)));
    }
    p->offset = 0;

    // ---- scratch sized for max_slices ----
    const long long cap = round_up(p->max_slices > 0 ? p->max_slices : kStepSlices, kStepSlices);
    long long zc = (long long)(kScratchBudget / ((size_t)B * K * sizeof(float2)));
    zc = zc / 1024 * 1024;
    if (zc < 1024) zc = 1024;
    p->zchunk = round_up(zc < cap ? zc : cap, 32);      // whole 32-slice tiles of the scratch layout
    if ((st = dev_alloc(p, &p->dZ, (size_t)B * K * p->zchunk)) != LOFAR_OK) return st;
    const long long nsteps = cap / kStepSlices;
    p->partial_pitch = (int)nsteps;
    p->chunkmax_pitch = nsteps;
    if ((st = dev_alloc(p, &p->dPartial, (size_t)ns * nsteps)) != LOFAR_OK) return st;
    if ((st = dev_alloc(p, &p->dChunkMax, (size_t)ns * nsteps)) != LOFAR_OK) return st;
    p->built = true;
    return LOFAR_OK;
}

lofar_status ensure(lofar_plan *p, int slices)
{
    if (!p) return LOFAR_E_INVALID;
    if (slices <= 0) return LOFAR_E_INVALID;
    if (p->max_slices <= 0) { p->max_slices = slices; p->built = false; }
    if (slices > p->max_slices) return LOFAR_E_SHAPE;
    if (!p->built) return build(p);
    return LOFAR_OK;
}

// Spans of the inverse-PPF launch: minimise (waves of CTAs) x (steps per span + warm-up step).
void plan_spans(long long nsteps, int nseries, int sms, int *nspans, int *span_len)
{
    long long best_cost = -1, best = 1;
    const long long lim = nsteps < 4096 ? nsteps : 4096;
    for (long long n = 1; n <= lim; ++n) {
        const long long per = (nsteps + n - 1) / n;
        const long long real = (nsteps + per - 1) / per;
        const long long waves = ((long long)nseries * real + sms - 1) / sms;
        const long long cost = waves * (per + (real > 1 ? 1 : 0));
        if (best_cost < 0 || cost < best_cost) { best_cost = cost; best = n; }
    }
    const long long per = (nsteps + best - 1) / best;
    *nspans = (int)((nsteps + per - 1) / per);
    *span_len = (int)(per * kStepSlices);
}

int beamform_dispatch(lofar_plan *p, const BeamformArgs &b, cudaStream_t st)
{
    if (p->dWimg && p->B >= p->tc_min_beams && tc_supported(b)) return launch_beamform_tc(b, p->dWimg, st);
    return launch_beamform(b, st);
}

lofar_status do_ippf(lofar_plan *p, const float2 *Z, long long zpitch, int ztile, long long nc, int zmap_trials,
                     float *series, long long series_pitch, long long out0, int *partial0, long long step0,
                     cudaStream_t st)
{
    IppfArgs a{};
    a.Z = Z; a.zpitch = zpitch; a.ztile = ztile; a.nc = nc;
    a.series = series; a.series_pitch = series_pitch; a.out0 = out0;
    a.Dph = p->dDph; a.zmap_trials = zmap_trials;
    a.K = p->K; a.k0 = p->k0; a.nseries = p->B * p->D;
    plan_spans((nc + kStepSlices - 1) / kStepSlices, a.nseries, p->num_sms, &a.nspans, &a.span_len);
    a.hist_in = p->dHist[p->hist_parity];
    a.hist_out = p->dHist[p->hist_parity ^ 1];
    a.gs = p->dGs; a.tw = p->dTw;
    a.partial = p->dPartial; a.partial_pitch = p->partial_pitch; a.partial0 = *partial0;
    a.chunkmax = p->dChunkMax; a.chunkmax_pitch = p->chunkmax_pitch; a.step0 = step0;
    a.vec_ok = ((zpitch & 1) == 0) && ((reinterpret_cast<size_t>(Z) & 15) == 0) &&
               (zpitch * (long long)p->K < (1LL << 32));   // 32-bit row offsets in the fast path
    ProfScope prof(p, 1, st);
    const int n = launch_ippf(a, st);
    if (n < 0) return LOFAR_E_CUDA;
    p->launches += n;
    p->hist_parity ^= 1;
    *partial0 += a.nspans;
    return LOFAR_OK;
}

TriggerArgs trigger_args(lofar_plan *p, const float *series, long long N, lofar_candidate *cand,
                         uint32_t *count, float *sigma)
{
    TriggerArgs t{};
    t.series = series; t.series_pitch = N; t.N = N;
    t.B = p->B; t.D = p->D; t.W = p->env_window; t.kappa = (float)p->kappa;
    t.tail = p->dTail;
    t.partial = p->dPartial; t.partial_pitch = p->partial_pitch;
    t.chunkmax = p->dChunkMax; t.chunkmax_pitch = p->chunkmax_pitch;
    t.nchunks = (N + 16383) / 16384;
    t.sigma = sigma; t.cand = cand; t.count = count; t.cap = p->max_cand;
    t.offset = p->offset;
    return t;
}

lofar_status check_x(const lofar_plan *p, const void *X, int slices)
{
    if (!X) return LOFAR_E_INVALID;
    const size_t pitch = (size_t)slices * sample_bytes(p);
    if ((reinterpret_cast<size_t>(X) & 15) || (pitch & 15)) return LOFAR_E_ALIGN;
    return LOFAR_OK;
}

lofar_status run_block_impl(lofar_plan *p, const void *X, int slices, float *series, lofar_candidate *cand,
                            uint32_t *count, float *sigma, cudaStream_t st)
{
    const long long T = slices, N = T * kMfft;
    int partial0 = 0;
    for (long long c0 = 0; c0 < T; c0 += p->zchunk) {
        const long long nc = (T - c0 < p->zchunk) ? T - c0 : p->zchunk;
        BeamformArgs b{};
        b.X = X; b.xpitch = T; b.t0 = c0; b.nt = nc;
        b.Z = p->dZ; b.zpitch = p->zchunk; b.ztile = 1;
        b.W = p->dW; b.Dph = p->dDph;
        b.S = p->S; b.K = p->K; b.B = p->B; b.nphase = 0; b.dtype = p->dtype;
        {
            ProfScope prof(p, 0, st);
            const int n = beamform_dispatch(p, b, st);
            if (n < 0) return LOFAR_E_CUDA;
            p->launches += n;
        }
        lofar_status s = do_ippf(p, p->dZ, p->zchunk, 1, nc, p->D > 1 ? p->D : 0, series, N, c0 * kMfft, &partial0,
                                 c0 / kStepSlices, st);
        if (s != LOFAR_OK) return s;
    }
    TriggerArgs t = trigger_args(p, series, N, cand, count, sigma);
    int n;
    ProfScope prof(p, 2, st);
    if (p->env_window == 1) {
        t.nparts = partial0;
    } else {
        t.nparts = (int)t.nchunks;
        if ((n = launch_trigger_reduce(t, st)) < 0) return LOFAR_E_CUDA;
        p->launches += n;
    }
    if ((n = launch_trigger_finish(t, st)) < 0) return LOFAR_E_CUDA;
    p->launches += n;
    if (p->env_window > 1) {
        if ((n = launch_tail_save(series, N, N, p->B * p->D, p->env_window, p->dTail, st)) < 0) return LOFAR_E_CUDA;
        p->launches += n;
    }
    p->offset += (uint64_t)N;
    return LOFAR_OK;
}

}  // namespace

// ================================================================================ C ABI
extern "C" {

lofar_status lofar_plan_create(lofar_plan **out, int stations, int subbands, int beams, int taps,
                               double stec_tecu)
{
    if (!out) return LOFAR_E_INVALID;
    *out = nullptr;
    if (stations <= 0 || subbands <= 0 || beams <= 0) return LOFAR_E_INVALID;
    if (taps != kTaps) return LOFAR_E_INVALID;
    if (subbands > kHalf) return LOFAR_E_SHAPE;
    lofar_plan *p = new (std::nothrow) lofar_plan();
    if (!p) return LOFAR_E_ALLOC;
    p->S = stations; p->K = subbands; p->B = beams; p->D = 1;
    p->tau.assign((size_t)beams * stations, 0.0);
    p->stec.assign(1, stec_tecu);
    default_prototype(p->h);
    *out = p;
    return LOFAR_OK;
}

void lofar_plan_destroy(lofar_plan *p)
{
    if (!p) return;
    if (p->s_copy) { cudaStreamSynchronize(p->s_copy); cudaStreamDestroy(p->s_copy); }
    if (p->s_comp) { cudaStreamSynchronize(p->s_comp); cudaStreamDestroy(p->s_comp); }
    for (int i = 0; i < 2; ++i) {
        if (p->ev_copied[i]) cudaEventDestroy(p->ev_copied[i]);
        if (p->ev_done[i]) cudaEventDestroy(p->ev_done[i]);
    }
    if (p->hCount) cudaFreeHost(p->hCount);
    for (auto &r : p->prof_pending) { cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
    for (auto e : p->prof_pool) cudaEventDestroy(e);
    free_tables(p);
    delete p;
}

lofar_status lofar_plan_set_band(lofar_plan *p, int first_subband, double f_zone_hz, double clock_hz,
                                 int fft_size)
{
    if (!p) return LOFAR_E_INVALID;
    if (fft_size != kMfft || !(clock_hz > 0.0) || !(f_zone_hz >= 0.0)) return LOFAR_E_INVALID;
    if (first_subband < 0 || first_subband + p->K > kHalf) return LOFAR_E_SHAPE;
    p->k0 = first_subband; p->f_zone = f_zone_hz; p->clock = clock_hz;
    p->built = false;
    return LOFAR_OK;
}

lofar_status lofar_plan_set_delays(lofar_plan *p, const double *tau)
{
    if (!p || !tau) return LOFAR_E_INVALID;
    p->tau.assign(tau, tau + (size_t)p->B * p->S);
    p->built = false;
    return LOFAR_OK;
}

lofar_status lofar_plan_set_trials(lofar_plan *p, int ntrials, const double *stec)
{
    if (!p || !stec || ntrials <= 0) return LOFAR_E_INVALID;
    p->D = ntrials;
    p->stec.assign(stec, stec + ntrials);
    p->built = false;
    return LOFAR_OK;
}

lofar_status lofar_plan_set_filter(lofar_plan *p, const double *h)
{
    if (!p) return LOFAR_E_INVALID;
    if (h) p->h.assign(h, h + (size_t)kMfft * kTaps);
    else default_prototype(p->h);
    p->built = false;
    return LOFAR_OK;
}

lofar_status lofar_plan_set_input(lofar_plan *p, lofar_dtype dtype, int max_slices)
{
    if (!p || max_slices <= 0) return LOFAR_E_INVALID;
    if (dtype != LOFAR_CI8 && dtype != LOFAR_CI16) return LOFAR_E_INVALID;
    p->dtype = dtype; p->max_slices = max_slices;
    p->built = false;
    return LOFAR_OK;
}

lofar_status lofar_plan_set_trigger(lofar_plan *p, double kappa, int env_window, uint32_t max_candidates)
{
    if (!p || !(kappa > 0.0) || env_window < 1 || env_window > 1024 || max_candidates == 0) return LOFAR_E_INVALID;
    p->kappa = kappa; p->env_window = env_window; p->max_cand = max_candidates;
    p->built = false;
    return LOFAR_OK;
}

lofar_status lofar_plan_workspace_bytes(lofar_plan *p, size_t *bytes)
{
    if (!p || !bytes) return LOFAR_E_INVALID;
    if (p->built) { *bytes = p->device_bytes; return LOFAR_OK; }
    // what build() will allocate for the current settings (streaming buffers excluded until used)
    const size_t ns = (size_t)p->B * p->D;
    const long long cap = round_up(p->max_slices > 0 ? p->max_slices : kStepSlices, kStepSlices);
    long long zc = (long long)(kScratchBudget / ((size_t)p->B * p->K * sizeof(float2))) / 1024 * 1024;
    if (zc < 1024) zc = 1024;
    if (zc > cap) zc = round_up(cap, 32);
    size_t b = 0;
    b += ((size_t)p->K * p->B * p->S + (size_t)p->D * p->K + (size_t)kTaps * kHalf + 768) * sizeof(float2);
    b += 2 * ns * (kTaps - 1) * kMfft * sizeof(float);
    b += ns * (size_t)(p->env_window - 1) * sizeof(float);
    b += (size_t)p->B * p->K * zc * sizeof(float2);
    b += ns * (size_t)(cap / kStepSlices) * (sizeof(double) + sizeof(float));
    *bytes = b;
    return LOFAR_OK;
}

lofar_status lofar_beamform_dedisperse(lofar_plan *p, const void *X, int slices, void *Z, void *stream)
{
    lofar_status s = ensure(p, slices);
    if (s != LOFAR_OK) return s;
    if (!Z) return LOFAR_E_INVALID;
    if ((s = check_x(p, X, slices)) != LOFAR_OK) return s;
    BeamformArgs b{};
    b.X = X; b.xpitch = slices; b.t0 = 0; b.nt = slices;
    b.Z = static_cast<float2 *>(Z); b.zpitch = slices; b.ztile = 0;
    b.W = p->dW; b.Dph = p->dDph;
    b.S = p->S; b.K = p->K; b.B = p->B; b.nphase = p->D > 1 ? p->D : 0; b.dtype = p->dtype;
    ProfScope prof(p, 0, static_cast<cudaStream_t>(stream));
    const int n = beamform_dispatch(p, b, static_cast<cudaStream_t>(stream));
    if (n < 0) return LOFAR_E_CUDA;
    p->launches += n;
    return LOFAR_OK;
}

lofar_status lofar_inverse_ppf(lofar_plan *p, const void *Z, int slices, float *series, void *stream)
{
    lofar_status s = ensure(p, slices);
    if (s != LOFAR_OK) return s;
    if (!Z || !series) return LOFAR_E_INVALID;
    if (reinterpret_cast<size_t>(Z) & 7 || reinterpret_cast<size_t>(series) & 7) return LOFAR_E_ALIGN;
    int partial0 = 0;
    return do_ippf(p, static_cast<const float2 *>(Z), slices, 0, slices, 0, series, (long long)slices * kMfft, 0,
                   &partial0, 0, static_cast<cudaStream_t>(stream));
}

lofar_status lofar_trigger(lofar_plan *p, const float *series, int slices, lofar_candidate *cand,
                           uint32_t *count, float *sigma, void *stream)
{
    lofar_status s = ensure(p, slices);
    if (s != LOFAR_OK) return s;
    if (!series || !cand || !count || !sigma) return LOFAR_E_INVALID;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const long long N = (long long)slices * kMfft;
    TriggerArgs t = trigger_args(p, series, N, cand, count, sigma);
    t.nparts = (int)t.nchunks;
    int n;
    ProfScope prof(p, 2, st);
    if ((n = launch_trigger_reduce(t, st)) < 0) return LOFAR_E_CUDA;
    p->launches += n;
    if ((n = launch_trigger_finish(t, st)) < 0) return LOFAR_E_CUDA;
    p->launches += n;
    if (p->env_window > 1) {
        if ((n = launch_tail_save(series, N, N, p->B * p->D, p->env_window, p->dTail, st)) < 0) return LOFAR_E_CUDA;
        p->launches += n;
    }
    p->offset += (uint64_t)N;
    return LOFAR_OK;
}

lofar_status lofar_run_block(lofar_plan *p, const void *X, int slices, float *series, lofar_candidate *cand,
                             uint32_t *count, float *sigma, void *stream)
{
    lofar_status s = ensure(p, slices);
    if (s != LOFAR_OK) return s;
    if (!series || !cand || !count || !sigma) return LOFAR_E_INVALID;
    if ((s = check_x(p, X, slices)) != LOFAR_OK) return s;
    return run_block_impl(p, X, slices, series, cand, count, sigma, static_cast<cudaStream_t>(stream));
}

lofar_status lofar_stream_reset(lofar_plan *p)
{
    if (!p) return LOFAR_E_INVALID;
    if (p->s_copy) CU(cudaStreamSynchronize(p->s_copy));
    if (p->s_comp) CU(cudaStreamSynchronize(p->s_comp));
    p->offset = 0;
    p->pushes = 0;
    p->slot_used[0] = p->slot_used[1] = false;
    if (p->built) {
        CU(cudaDeviceSynchronize());
        const size_t hist = (size_t)p->B * p->D * (kTaps - 1) * kMfft * sizeof(float);
        CU(cudaMemset(p->dHist[0], 0, hist));
        CU(cudaMemset(p->dHist[1], 0, hist));
        if (p->dTail) CU(cudaMemset(p->dTail, 0, (size_t)p->B * p->D * (p->env_window - 1) * sizeof(float)));
        CU(cudaDeviceSynchronize());
    }
    return LOFAR_OK;
}

lofar_status lofar_stream_push(lofar_plan *p, const void *X_host, int slices, float *series,
                               lofar_candidate *cand_host, uint32_t *count_host, float *sigma_host)
{
    lofar_status s = ensure(p, slices);
    if (s != LOFAR_OK) return s;
    if (!X_host || !series) return LOFAR_E_INVALID;
    if (((size_t)slices * sample_bytes(p)) & 15) return LOFAR_E_ALIGN;
    if (p->pushes >= kCountRing) return LOFAR_E_STATE;   // call lofar_stream_sync at least every 64 pushes
    const int ns = p->B * p->D;
    if (!p->s_copy) {
        CU(cudaStreamCreateWithFlags(&p->s_copy, cudaStreamNonBlocking));
        CU(cudaStreamCreateWithFlags(&p->s_comp, cudaStreamNonBlocking));
        for (int i = 0; i < 2; ++i) {
            CU(cudaEventCreateWithFlags(&p->ev_copied[i], cudaEventDisableTiming));
            CU(cudaEventCreateWithFlags(&p->ev_done[i], cudaEventDisableTiming));
        }
        CU(cudaMallocHost(reinterpret_cast<void **>(&p->hCount), kCountRing * sizeof(uint32_t)));
    }
    if (!p->dX[0]) {
        const size_t bytes = (size_t)p->S * 2 * p->K * (size_t)p->max_slices * sample_bytes(p);
        for (int i = 0; i < 2; ++i) {
            char *x = nullptr;
            if ((s = dev_alloc(p, &x, bytes)) != LOFAR_OK) return s;
            p->dX[i] = x;
            if ((s = dev_alloc(p, &p->dCand[i], (size_t)p->max_cand)) != LOFAR_OK) return s;
            if ((s = dev_alloc(p, &p->dCount[i], 1)) != LOFAR_OK) return s;
            if ((s = dev_alloc(p, &p->dSigma[i], (size_t)ns)) != LOFAR_OK) return s;
        }
        p->dX_bytes = bytes;
    }
    const int slot = (int)(p->push_index & 1);
    const size_t bytes = (size_t)p->S * 2 * p->K * (size_t)slices * sample_bytes(p);
    if (p->slot_used[slot]) CU(cudaStreamWaitEvent(p->s_copy, p->ev_done[slot], 0));
    CU(cudaMemcpyAsync(p->dX[slot], X_host, bytes, cudaMemcpyHostToDevice, p->s_copy));
    CU(cudaEventRecord(p->ev_copied[slot], p->s_copy));
    CU(cudaStreamWaitEvent(p->s_comp, p->ev_copied[slot], 0));
    s = run_block_impl(p, p->dX[slot], slices, series, p->dCand[slot], p->dCount[slot], p->dSigma[slot], p->s_comp);
    if (s != LOFAR_OK) return s;
    CU(cudaMemcpyAsync(&p->hCount[p->pushes], p->dCount[slot], sizeof(uint32_t), cudaMemcpyDeviceToHost, p->s_comp));
    if (count_host)
        CU(cudaMemcpyAsync(count_host, p->dCount[slot], sizeof(uint32_t), cudaMemcpyDeviceToHost, p->s_comp));
    if (sigma_host)
        CU(cudaMemcpyAsync(sigma_host, p->dSigma[slot], (size_t)ns * sizeof(float), cudaMemcpyDeviceToHost, p->s_comp));
    if (cand_host)
        CU(cudaMemcpyAsync(cand_host, p->dCand[slot], (size_t)p->max_cand * sizeof(lofar_candidate),
                           cudaMemcpyDeviceToHost, p->s_comp));
    CU(cudaEventRecord(p->ev_done[slot], p->s_comp));
    p->slot_used[slot] = true;
    p->push_index++;
    p->pushes++;
    return LOFAR_OK;
}

lofar_status lofar_stream_sync(lofar_plan *p)
{
    if (!p) return LOFAR_E_INVALID;
    if (p->s_copy) CU(cudaStreamSynchronize(p->s_copy));
    if (p->s_comp) CU(cudaStreamSynchronize(p->s_comp));
    bool over = false;
    for (int i = 0; i < p->pushes; ++i) over = over || (p->hCount[i] > p->max_cand);
    p->pushes = 0;
    return over ? LOFAR_E_OVERFLOW : LOFAR_OK;
}

lofar_status lofar_plan_profile(lofar_plan *p, int enable)
{
    if (!p) return LOFAR_E_INVALID;
    p->prof = enable != 0;
    return LOFAR_OK;
}

lofar_status lofar_plan_profile_read(lofar_plan *p, double *ms, uint64_t *launches)
{
    if (!p || !ms || !launches) return LOFAR_E_INVALID;
    for (auto &r : p->prof_pending) {
        float t = 0.f;
        CU(cudaEventSynchronize(r.b));
        CU(cudaEventElapsedTime(&t, r.a, r.b));
        if (r.id >= 0 && r.id < 3) { ms[r.id] += (double)t; launches[r.id] += 1; }
        p->prof_pool.push_back(r.a);
        p->prof_pool.push_back(r.b);
    }
    p->prof_pending.clear();
    return LOFAR_OK;
}

uint64_t lofar_plan_launch_count(const lofar_plan *p) { return p ? p->launches : 0; }

const char *lofar_status_string(lofar_status s)
{
    switch (s) {
    case LOFAR_OK: return "ok";
    case LOFAR_E_INVALID: return "invalid argument";
    case LOFAR_E_SHAPE: return "shape out of range";
    case LOFAR_E_ALIGN: return "pointer or row pitch not aligned";
    case LOFAR_E_ALLOC: return "allocation failed";
    case LOFAR_E_CUDA: return "CUDA error";
    case LOFAR_E_OVERFLOW: return "candidate buffer overflow";
    case LOFAR_E_STATE: return "illegal call in this state";
    }
    return "unknown status";
}

}  // extern "C"
