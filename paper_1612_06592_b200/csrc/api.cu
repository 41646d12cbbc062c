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
    if (p->alloc_fn) {
        v = p->alloc_fn(count * sizeof(T), p->alloc_ctx);
        if (!v) return LOFAR_E_ALLOC;
    } else {
        cudaError_t e = cudaMalloc(&v, count * sizeof(T));
        if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); return LOFAR_E_ALLOC; }
        if (e != cudaSuccess) return LOFAR_E_CUDA;
    }
    *ptr = static_cast<T *>(v);
    p->device_bytes += count * sizeof(T);
    return LOFAR_OK;
}

template <typename T>
void dev_free(lofar_plan *p, T *&ptr)
{
    if (ptr) {
        if (p->free_fn) p->free_fn(const_cast<void *>(static_cast<const void *>(ptr)), p->alloc_ctx);
        else cudaFree(const_cast<void *>(static_cast<const void *>(ptr)));
    }
    ptr = nullptr;
}

void free_staging(lofar_plan *p)
{
    for (int i = 0; i < 2; ++i) {
        char *x = static_cast<char *>(p->dX[i]);
        dev_free(p, x);
        p->dX[i] = nullptr;
        dev_free(p, p->dCand[i]); dev_free(p, p->dCount[i]); dev_free(p, p->dSigma[i]);
    }
    p->dX_bytes = 0;
}

// Waits for the plan's own streams; buffers may then be released (caller streams are the caller's to order).
void quiesce(lofar_plan *p)
{
    if (p->s_copy) cudaStreamSynchronize(p->s_copy);
    if (p->s_comp) cudaStreamSynchronize(p->s_comp);
    if (p->s_bf) cudaStreamSynchronize(p->s_bf);
    if (p->s_ippf) cudaStreamSynchronize(p->s_ippf);
}

// SMs the inverse-PPF spans are planned for: with the two-lane pipeline a few SMs are left to the beamformer
// (an inverse-PPF CTA owns the whole register file and shared memory of its SM, so nothing co-resides with it).
int ippf_sm_budget(int num_sms, bool overlap)
{
    if (!overlap) return num_sms;
    const int keep = num_sms - 16;
    return keep > num_sms / 2 ? keep : num_sms / 2;
}

void free_tables(lofar_plan *p)
{
    quiesce(p);
    dev_free(p, p->dWimg);
    dev_free(p, p->dW); dev_free(p, p->dDph); dev_free(p, p->dGs); dev_free(p, p->dTw);
    dev_free(p, p->dHist[0]); dev_free(p, p->dHist[1]); dev_free(p, p->dTail);
    dev_free(p, p->dZ); dev_free(p, p->dPartial); dev_free(p, p->dChunkMax);
    dev_free(p, p->dXhat); dev_free(p, p->dDtab); dev_free(p, p->dTw8192); dev_free(p, p->dTw16k);
    dev_free(p, p->dY); dev_free(p, p->dLsmrWork); dev_free(p, p->dLsmrPartial);
    { char *sc = static_cast<char *>(p->dLsmrScal); dev_free(p, sc); p->dLsmrScal = nullptr; }
    dev_free(p, p->dItems); dev_free(p, p->dNItems); dev_free(p, p->dSigmaRef); dev_free(p, p->dThr); dev_free(p, p->dHist0);
    p->have_ref = false;
    free_staging(p);
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

// Element counts of every plan-owned device buffer for the current settings: build() allocates exactly
// these, lofar_plan_workspace_bytes reports their sum.
struct Layout {
    bool tc;                 // tensor-core operand images wanted (int8 input)
    size_t W, Dph, gs, tw, wimg, hist, tail, Z, partial, chunkmax, items;
    size_t y, lsmr_work, lsmr_scal_bytes, lsmr_partial;   // LSMR inversion only
    long long ypitch, wpitch;
    size_t xhat, dtab, tw8192, tw16k;  // exact de-dispersion only
    long long xhat_pitch;
    size_t x_bytes, cand, sigma;   // streaming staging (per slot)
    long long cap, zchunk, nsteps;
    bool overlap;            // two-lane pipeline: two scratch slots of zchunk slices each
    size_t table_bytes() const
    {
        return (W + Dph + gs + tw + Z) * sizeof(float2) + wimg * sizeof(unsigned short) +
               (3 * hist + tail + chunkmax + 2 * sigma) * sizeof(float) + partial * sizeof(double) +
               items * sizeof(int2) + sizeof(uint32_t) +
               (y + lsmr_work + xhat) * sizeof(float) + lsmr_scal_bytes + lsmr_partial * sizeof(double) +
               (dtab + tw8192 + tw16k) * sizeof(float2);
    }
    size_t staging_bytes() const
    {
        return 2 * (x_bytes + cand * sizeof(lofar_candidate) + sizeof(uint32_t) + sigma * sizeof(float));
    }
};

Layout layout(const lofar_plan *p)
{
    Layout L{};
    const size_t S = p->S, K = p->K, B = p->B, D = p->D, ns = B * D, ni = (size_t)p->ninv();
    L.tc = p->dtype == LOFAR_CI8 && p->S <= 32 && p->B <= 128;
    L.W = K * B * S; L.Dph = D * K; L.gs = (size_t)kTaps * kHalf; L.tw = 256 + 512;
    L.wimg = L.tc ? K * 2 * tc_image_halfs(p->S, p->B) : 0;
    L.hist = ni * (kTaps - 1) * kMfft;
    L.tail = ns * (size_t)(p->env_window - 1);
    L.cap = round_up(p->max_slices > 0 ? p->max_slices : kStepSlices, kStepSlices);
    long long zc = (long long)(p->scratch_limit / (B * K * sizeof(float2)));
    zc = zc >= 1024 ? zc / 1024 * 1024 : zc / 32 * 32;
    if (zc < 32) zc = 32;
    // Two-lane pipeline: only with the tensor-core beamformer (a few SMs keep it at its HBM rate) and only if the
    // block then has at least two chunks; the two slots share the scratch budget.
    L.overlap = p->overlap != 0 && L.tc && p->B >= p->tc_min_beams;
    if (L.overlap) {
        long long zo = zc / 2;
        if (zo > p->overlap_chunk) zo = p->overlap_chunk;
        zo = zo >= 1024 ? zo / 1024 * 1024 : zo / 32 * 32;
        if (zo < 32 || L.cap <= zo) L.overlap = false;     // a single chunk: nothing to pipeline
        else zc = zo;
    }
    L.zchunk = round_up(zc < L.cap ? zc : L.cap, 32);      // whole 32-slice tiles of the scratch layout
    L.Z = B * K * (size_t)L.zchunk * (L.overlap ? 2 : 1);
    L.nsteps = L.cap / kStepSlices;
    L.partial = ns * (size_t)L.nsteps;
    L.chunkmax = ns * (size_t)L.nsteps;
    L.items = 16384;                   // flagged chunks per block before the scan falls back to all of them
    if (p->inversion == LOFAR_INV_LSMR) {
        const long long T = p->max_slices > 0 ? p->max_slices : kStepSlices;
        L.ypitch = (T + kTaps - 1) * kMfft;
        L.wpitch = (T + 2 * (kTaps - 1)) * kMfft;
        L.y = ni * (size_t)L.ypitch;
        L.lsmr_work = 4 * ni * (size_t)L.wpitch;
        L.lsmr_scal_bytes = lsmr_scalar_bytes((int)ni);
        L.lsmr_partial = lsmr_partial_count((int)ni, T + 2 * (kTaps - 1));
    }
    if (p->dedisp == LOFAR_DEDISP_EXACT) {
        const long long T = p->max_slices > 0 ? p->max_slices : kStepSlices;
        L.xhat_pitch = (T + 2) * kMfft;
        L.xhat = B * (size_t)L.xhat_pitch;
        L.dtab = D * (size_t)8193; L.tw8192 = 8192; L.tw16k = 4097;
    }
    L.x_bytes = S * 2 * K * (size_t)(p->max_slices > 0 ? p->max_slices : 0) * sample_bytes(p);
    L.cand = p->max_cand; L.sigma = ns;
    return L;
}

// Causal sigma: the reference level a stream starts with (lofar_plan_set_sigma_mode).
lofar_status load_sigma_init(lofar_plan *p, cudaStream_t st)
{
    p->have_ref = false;
    const size_t ns = (size_t)p->B * p->D;
    if (p->sigma_mode != LOFAR_SIGMA_CAUSAL || p->sigma_init.size() != ns) return LOFAR_OK;
    p->thr_init.resize(ns);
    for (size_t i = 0; i < ns; ++i) p->thr_init[i] = (float)p->kappa * p->sigma_init[i];
    // the host vectors live in the plan, so the stream-ordered copies may read them later
    CU(cudaMemcpyAsync(p->dSigmaRef, p->sigma_init.data(), ns * sizeof(float), cudaMemcpyHostToDevice, st));
    CU(cudaMemcpyAsync(p->dThr, p->thr_init.data(), ns * sizeof(float), cudaMemcpyHostToDevice, st));
    p->have_ref = true;
    return LOFAR_OK;
}

lofar_status build(lofar_plan *p)
{
    free_tables(p);
    int dev = 0;
    CU(cudaGetDevice(&dev));
    CU(cudaDeviceGetAttribute(&p->num_sms, cudaDevAttrMultiProcessorCount, dev));
    if (ippf_configure() != 0) return LOFAR_E_CUDA;
    const Layout L = layout(p);
    if (L.tc && tc_configure() != 0) return LOFAR_E_CUDA;
    const int S = p->S, K = p->K, B = p->B, D = p->D;

    // ---- tables, in double on the host, rounded once to fp32 ----
    std::vector<float2> W(L.W), Dph(L.Dph), gs(L.gs), tw(L.tw);
    const bool tc = L.tc;
    const size_t img = tc ? tc_image_halfs(S, B) : 0;
    std::vector<unsigned short> wimg(L.wimg);
    std::vector<double> wre((size_t)B * S), wim((size_t)B * S);
    for (int j = 0; j < K; ++j) {
        const double f = p->f_zone + (double)(p->k0 + j) * (p->clock / kMfft);
        for (int d = 0; d < D; ++d) Dph[(size_t)d * K + j] = unit_phasor(-(kDispersion * p->stec[d] / f));
        // one trial: fold the phase into W (not in exact mode, where the series is de-dispersed after the inversion)
        const double fold = (D == 1 && p->dedisp != LOFAR_DEDISP_EXACT) ? -(kDispersion * p->stec[0] / f) : 0.0;
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
    // twiddles: w1024[256] for the pre-pass, TBs[r][j] = +-exp(2 pi i j r / 512) (r < 32, j < 16) for the radix-32 pass
    for (int m = 0; m < 256; ++m) tw[m] = unit_phasor((double)m / 1024.0);
    // the odd rows carry the sign (-1)^((r-1)/2): it rotates the odd half of the radix-32 butterflies by 8 outputs, which
    // lets the two lanes of a butterfly exchange half as many registers (fft_warp.cuh: fft512_pass_b)
    for (int r = 0; r < 32; ++r)
        for (int jj = 0; jj < 16; ++jj) {
            float2 v = unit_phasor((double)(jj * r) / 512.0);
            if ((r & 3) == 3) { v.x = -v.x; v.y = -v.y; }
            tw[256 + r * 16 + jj] = v;
        }

    lofar_status st;
    if ((st = dev_alloc(p, &p->dW, L.W)) != LOFAR_OK) return st;
    if ((st = dev_alloc(p, &p->dDph, L.Dph)) != LOFAR_OK) return st;
    if ((st = dev_alloc(p, &p->dGs, L.gs)) != LOFAR_OK) return st;
    if ((st = dev_alloc(p, &p->dTw, L.tw)) != LOFAR_OK) return st;
    if (tc) {
        if ((st = dev_alloc(p, &p->dWimg, L.wimg)) != LOFAR_OK) return st;
        CU(cudaMemcpy(p->dWimg, wimg.data(), wimg.size() * sizeof(unsigned short), cudaMemcpyHostToDevice));
    }
    CU(cudaMemcpy(p->dW, W.data(), W.size() * sizeof(float2), cudaMemcpyHostToDevice));
    CU(cudaMemcpy(p->dDph, Dph.data(), Dph.size() * sizeof(float2), cudaMemcpyHostToDevice));
    CU(cudaMemcpy(p->dGs, gs.data(), gs.size() * sizeof(float2), cudaMemcpyHostToDevice));
    CU(cudaMemcpy(p->dTw, tw.data(), tw.size() * sizeof(float2), cudaMemcpyHostToDevice));

    // ---- carried state ----
    for (int i = 0; i < 2; ++i) {
        if ((st = dev_alloc(p, &p->dHist[i], L.hist)) != LOFAR_OK) return st;
        CU(cudaMemset(p->dHist[i], 0, L.hist * sizeof(float)));
    }
    p->hist_parity = 0;
    if (L.tail) {
        if ((st = dev_alloc(p, &p->dTail, L.tail)) != LOFAR_OK) return st;
        CU(cudaMemset(p->dTail, 0, L.tail * sizeof(float)));
    }
    p->offset = 0;
    p->reset_pending = false;

    // ---- scratch sized for max_slices ----
    p->zchunk = L.zchunk;
    p->overlap_on = L.overlap;
    p->ippf_sms = ippf_sm_budget(p->num_sms, L.overlap);
    if (L.overlap && !p->s_bf) {
        // the inverse PPF goes first wherever both kernels have CTAs pending; the beamformer fills what is left
        int least = 0, greatest = 0;
        CU(cudaDeviceGetStreamPriorityRange(&least, &greatest));
        CU(cudaStreamCreateWithPriority(&p->s_ippf, cudaStreamNonBlocking, greatest));
        CU(cudaStreamCreateWithPriority(&p->s_bf, cudaStreamNonBlocking, least));
        CU(cudaEventCreateWithFlags(&p->ev_fork, cudaEventDisableTiming));
        CU(cudaEventCreateWithFlags(&p->ev_join, cudaEventDisableTiming));
        for (int i = 0; i < 2; ++i) {
            CU(cudaEventCreateWithFlags(&p->ev_bf[i], cudaEventDisableTiming));
            CU(cudaEventCreateWithFlags(&p->ev_ippf[i], cudaEventDisableTiming));
        }
    }
    if ((st = dev_alloc(p, &p->dZ, L.Z)) != LOFAR_OK) return st;
    CU(cudaMemset(p->dZ, 0, L.Z * sizeof(float2)));
    p->partial_pitch = (int)L.nsteps;
    p->chunkmax_pitch = L.nsteps;
    if ((st = dev_alloc(p, &p->dPartial, L.partial)) != LOFAR_OK) return st;
    if ((st = dev_alloc(p, &p->dChunkMax, L.chunkmax)) != LOFAR_OK) return st;
    p->items_cap = (uint32_t)L.items;
    if ((st = dev_alloc(p, &p->dItems, L.items)) != LOFAR_OK) return st;
    if ((st = dev_alloc(p, &p->dNItems, 1)) != LOFAR_OK) return st;
    if ((st = dev_alloc(p, &p->dSigmaRef, L.sigma)) != LOFAR_OK) return st;
    if ((st = dev_alloc(p, &p->dThr, L.sigma)) != LOFAR_OK) return st;
    if ((st = dev_alloc(p, &p->dHist0, L.hist)) != LOFAR_OK) return st;
    CU(cudaMemset(p->dNItems, 0, sizeof(uint32_t)));
    if (p->dedisp == LOFAR_DEDISP_EXACT) {
        if (dedisp_configure() != 0) return LOFAR_E_CUDA;
        p->xhat_pitch = L.xhat_pitch;
        if ((st = dev_alloc(p, &p->dXhat, L.xhat)) != LOFAR_OK) return st;
        CU(cudaMemset(p->dXhat, 0, L.xhat * sizeof(float)));
        std::vector<float2> dt(L.dtab), t8(L.tw8192), t16(L.tw16k);
        const int nfft = 16 * kMfft;
        for (int d = 0; d < D; ++d)
            for (int j = 0; j <= nfft / 2; ++j) {
                const double fj = p->f_zone + (double)j * (p->clock / nfft);
                float2 v = unit_phasor(-(kDispersion * p->stec[d] / fj));
                if (j == 0 || j == nfft / 2) v.y = 0.f;         // the self-conjugate bins keep the real part
                dt[(size_t)d * 8193 + j] = v;
            }
        for (int m = 0; m < 8192; ++m) t8[m] = unit_phasor((double)m / 8192.0);
        for (int j = 0; j <= 4096; ++j) t16[j] = unit_phasor((double)j / 16384.0);
        if ((st = dev_alloc(p, &p->dDtab, L.dtab)) != LOFAR_OK) return st;
        if ((st = dev_alloc(p, &p->dTw8192, L.tw8192)) != LOFAR_OK) return st;
        if ((st = dev_alloc(p, &p->dTw16k, L.tw16k)) != LOFAR_OK) return st;
        CU(cudaMemcpy(p->dDtab, dt.data(), dt.size() * sizeof(float2), cudaMemcpyHostToDevice));
        CU(cudaMemcpy(p->dTw8192, t8.data(), t8.size() * sizeof(float2), cudaMemcpyHostToDevice));
        CU(cudaMemcpy(p->dTw16k, t16.data(), t16.size() * sizeof(float2), cudaMemcpyHostToDevice));
    }
    if (p->inversion == LOFAR_INV_LSMR) {
        p->ypitch = L.ypitch; p->wpitch = L.wpitch;
        if ((st = dev_alloc(p, &p->dY, L.y)) != LOFAR_OK) return st;
        if ((st = dev_alloc(p, &p->dLsmrWork, L.lsmr_work)) != LOFAR_OK) return st;
        char *sc = nullptr;
        if ((st = dev_alloc(p, &sc, L.lsmr_scal_bytes)) != LOFAR_OK) return st;
        p->dLsmrScal = sc;
        if ((st = dev_alloc(p, &p->dLsmrPartial, L.lsmr_partial)) != LOFAR_OK) return st;
    }
    if ((st = load_sigma_init(p, nullptr)) != LOFAR_OK) return st;
    CU(cudaDeviceSynchronize());       // build is the one place that may block: tables are in place when it returns
    p->built = true;
    return LOFAR_OK;
}

// Zeroes the carried state on the stream of the compute call that follows a lofar_stream_reset.
lofar_status apply_reset(lofar_plan *p, cudaStream_t st)
{
    if (!p->reset_pending) return LOFAR_OK;
    const size_t hist = (size_t)p->ninv() * (kTaps - 1) * kMfft * sizeof(float);
    CU(cudaMemsetAsync(p->dHist[0], 0, hist, st));
    CU(cudaMemsetAsync(p->dHist[1], 0, hist, st));
    if (p->dXhat)
        CU(cudaMemset2DAsync(p->dXhat, (size_t)p->xhat_pitch * sizeof(float), 0, 2 * kMfft * sizeof(float), (size_t)p->B, st));
    if (p->dTail) CU(cudaMemsetAsync(p->dTail, 0, (size_t)p->B * p->D * (p->env_window - 1) * sizeof(float), st));
    p->reset_pending = false;
    return load_sigma_init(p, st);
}

lofar_status ensure(lofar_plan *p, int slices)
{
    if (!p) return LOFAR_E_INVALID;
    if (slices <= 0) return LOFAR_E_INVALID;
    if (p->max_slices <= 0) { p->max_slices = slices; p->built = false; }
    if (slices > p->max_slices) return LOFAR_E_STATE;   // capacity fixed by lofar_plan_set_input
    if (!p->built) {
        const lofar_status st = build(p);
        if (st != LOFAR_OK) { free_tables(p); return st; }
    }
    return LOFAR_OK;
}

// Spans of the inverse-PPF launch: minimise (waves of CTAs) x (steps per span + warm-up step). one_wave: at most
// `sms` CTAs (the two-lane pipeline leaves the other SMs to the beamformer for the whole launch).
void plan_spans(long long nsteps, int nseries, int sms, bool one_wave, int *nspans, int *span_len)
{
    long long best_cost = -1, best = 1;
    long long lim = nsteps < 4096 ? nsteps : 4096;
    if (one_wave && nseries <= sms && lim > sms / nseries) lim = sms / nseries;
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

// LSMR inversion (f1): the carried 15 slices of y go in front of the rows the inverse DFT is about to write.
lofar_status lsmr_begin(lofar_plan *p, cudaStream_t st)
{
    const size_t row = (size_t)(kTaps - 1) * kMfft * sizeof(float);
    CU(cudaMemcpy2DAsync(p->dY, (size_t)p->ypitch * sizeof(float), p->dHist[p->hist_parity], row, row,
                         (size_t)p->ninv(), cudaMemcpyDeviceToDevice, st));
    return LOFAR_OK;
}

lofar_status lsmr_solve(lofar_plan *p, long long T, float *series, long long series_pitch, cudaStream_t st)
{
    ProfScope prof(p, 3, st);
    const int n = launch_lsmr(p->dY, p->ypitch, T, p->dLsmrWork, p->wpitch, reinterpret_cast<const float *>(p->dGs),
                              p->dLsmrScal, p->dLsmrPartial, p->ninv(), p->lsmr_iters, series, series_pitch, st);
    if (n < 0) return LOFAR_E_CUDA;
    p->launches += n;
    return LOFAR_OK;
}

// True while a block call runs its chunks through the two-lane pipeline (set by run_block_impl).
bool lanes_now(const lofar_plan *p, long long) { return p->lanes_active; }

struct EmitTo { lofar_candidate *cand; uint32_t *count; };   // cand == nullptr: no emission from the epilogue

lofar_status do_ippf(lofar_plan *p, const float2 *Z, long long zpitch, int ztile, long long nc, int zmap_trials,
                     float *series, long long series_pitch, long long out0, int *partial0, long long step0,
                     cudaStream_t st, EmitTo em = EmitTo{nullptr, nullptr}, bool y_only = false)
{
    IppfArgs a{};
    a.D = p->D; a.offset = p->offset;
    if (y_only) { a.yout = p->dY + (kTaps - 1) * kMfft; a.yout_pitch = p->ypitch; }
    if (em.cand) {
        a.thr = p->dThr; a.sigma_ref = p->dSigmaRef;
        a.cand = em.cand; a.count = em.count; a.cap = p->max_cand;
    }
    a.Z = Z; a.zpitch = zpitch; a.ztile = ztile; a.nc = nc;
    a.series = series; a.series_pitch = series_pitch; a.out0 = out0;
    a.Dph = p->dDph; a.zmap_trials = zmap_trials;
    a.K = p->K; a.k0 = p->k0; a.nseries = p->ninv();
    const bool lanes = ztile && lanes_now(p, nc);
    plan_spans((nc + kStepSlices - 1) / kStepSlices, a.nseries, lanes ? p->ippf_sms : p->num_sms, lanes, &a.nspans,
               &a.span_len);
    a.hist_in = p->dHist[p->hist_parity];
    a.hist_out = p->dHist[p->hist_parity ^ 1];
    a.gs = p->dGs; a.tw = p->dTw;
    a.partial = p->dPartial; a.partial_pitch = p->partial_pitch; a.partial0 = *partial0;
    a.chunkmax = p->dChunkMax; a.chunkmax_pitch = p->chunkmax_pitch; a.step0 = step0;
    a.vec_ok = ((zpitch & 1) == 0) && ((reinterpret_cast<size_t>(Z) & 15) == 0);
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
    t.sigma_thr = (p->sigma_mode == LOFAR_SIGMA_CAUSAL && p->have_ref) ? p->dSigmaRef : sigma;
    t.zero_count = 1;
    t.items = p->dItems; t.nitems = p->dNItems; t.items_cap = p->items_cap;
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
    const int ns = p->B * p->D;
    const bool causal = p->sigma_mode == LOFAR_SIGMA_CAUSAL;
    // how the candidates of this block are found:
    //   emit   -- threshold known before the block: decided in the inverse-PPF epilogue;
    //   scan   -- two-pass: sigma of this block, then the stored series is re-read where its maximum allows;
    //   rescan -- two-pass without a series: those places are recomputed from X.
    const bool lsmr = p->inversion == LOFAR_INV_LSMR, exact = p->dedisp == LOFAR_DEDISP_EXACT;
    const bool emit = causal && p->have_ref && !lsmr && !exact;   // LSMR / exact series are thresholded afterwards
    if (exact && series == nullptr) return LOFAR_E_INVALID;
    // exact de-dispersion: the inversion writes the undispersed series of each beam behind its two carried slices
    float *inv_series = exact ? p->dXhat + 2 * kMfft : series;
    const long long inv_pitch = exact ? p->xhat_pitch : N;
    const int ztrials = (p->D > 1 && !exact) ? p->D : 0;
    const bool rescan = !emit && series == nullptr;
    if ((causal || series == nullptr) && p->env_window != 1) return LOFAR_E_INVALID;
    if (lsmr && series == nullptr) return LOFAR_E_INVALID;
    if (lsmr) { const lofar_status s0 = lsmr_begin(p, st); if (s0 != LOFAR_OK) return s0; }
    if (emit || rescan) CU(cudaMemsetAsync(count, 0, sizeof(uint32_t), st));
    if (rescan)
        CU(cudaMemcpyAsync(p->dHist0, p->dHist[p->hist_parity], (size_t)ns * (kTaps - 1) * kMfft * sizeof(float),
                           cudaMemcpyDeviceToDevice, st));
    int partial0 = 0;
    // Chunk loop. Serial: both kernels of every chunk on the caller's stream. Two-lane pipeline (overlap_on): the
    // beamformer of chunk c + 1 runs on s_bf while the inverse PPF of chunk c runs on s_ippf; the two alternate
    // between the two scratch slots, chained by events; the caller's stream forks before and joins after the loop.
    const bool lanes = p->overlap_on && T > p->zchunk;
    p->lanes_active = lanes;
    cudaStream_t sb = lanes ? p->s_bf : st, si = lanes ? p->s_ippf : st;
    if (lanes) {
        CU(cudaEventRecord(p->ev_fork, st));
        CU(cudaStreamWaitEvent(sb, p->ev_fork, 0));
        CU(cudaStreamWaitEvent(si, p->ev_fork, 0));
    }
    const size_t zslot = (size_t)p->B * p->K * (size_t)p->zchunk;
    int ci = 0;
    for (long long c0 = 0; c0 < T; c0 += p->zchunk, ++ci) {
        const long long nc = (T - c0 < p->zchunk) ? T - c0 : p->zchunk;
        const int slot = lanes ? (ci & 1) : 0;
        float2 *Zc = p->dZ + (size_t)slot * zslot;
        BeamformArgs b{};
        b.X = X; b.xpitch = T; b.t0 = c0; b.nt = nc;
        b.Z = Zc; b.zpitch = p->zchunk; b.ztile = 1;
        b.W = p->dW; b.Dph = p->dDph;
        b.S = p->S; b.K = p->K; b.B = p->B; b.nphase = 0; b.dtype = p->dtype;
        if (lanes && ci >= 2) CU(cudaStreamWaitEvent(sb, p->ev_ippf[slot], 0));   // the slot has been consumed
        {
            ProfScope prof(p, 0, sb);
            const int n = beamform_dispatch(p, b, sb);
            if (n < 0) return LOFAR_E_CUDA;
            p->launches += n;
        }
        if (lanes) {
            CU(cudaEventRecord(p->ev_bf[slot], sb));
            CU(cudaStreamWaitEvent(si, p->ev_bf[slot], 0));
        }
        lofar_status s = do_ippf(p, Zc, p->zchunk, 1, nc, ztrials, lsmr ? nullptr : inv_series, inv_pitch, c0 * kMfft,
                                 &partial0, c0 / kStepSlices, si, emit ? EmitTo{cand, count} : EmitTo{nullptr, nullptr},
                                 lsmr);
        if (s != LOFAR_OK) return s;
        if (lanes) CU(cudaEventRecord(p->ev_ippf[slot], si));
    }
    if (lanes) {
        CU(cudaEventRecord(p->ev_join, si));                 // every beamformer launch has been waited for by s_ippf
        CU(cudaStreamWaitEvent(st, p->ev_join, 0));
    }
    if (lsmr) { const lofar_status s1 = lsmr_solve(p, T, inv_series, inv_pitch, st); if (s1 != LOFAR_OK) return s1; }
    if (exact) {
        DedispArgs d{};
        d.xlead = p->dXhat; d.xpitch = p->xhat_pitch; d.nlead = T + 2;
        d.series = series; d.series_pitch = N; d.T = T; d.B = p->B; d.D = p->D;
        d.Dtab = p->dDtab; d.tw8192 = p->dTw8192; d.tw16k = p->dTw16k; d.tw512 = p->dTw + 256;
        int nd;
        {
            ProfScope prof(p, 4, st);
            nd = launch_dedisp(d, st);
        }
        if (nd < 0) return LOFAR_E_CUDA;
        p->launches += nd;
        // carry the last two slices of the undispersed series (one slice at a time: they may overlap their target)
        for (int i = 0; i < 2; ++i)
            CU(cudaMemcpy2DAsync(p->dXhat + (size_t)i * kMfft, (size_t)p->xhat_pitch * sizeof(float),
                                 p->dXhat + (size_t)(T + i) * kMfft, (size_t)p->xhat_pitch * sizeof(float),
                                 kMfft * sizeof(float), (size_t)p->B, cudaMemcpyDeviceToDevice, st));
    }
    TriggerArgs t = trigger_args(p, series, N, cand, count, sigma);
    t.zero_count = (emit || rescan) ? 0 : 1;
    int n;
    ProfScope prof(p, 2, st);
    if (p->env_window == 1 && !lsmr && !exact) {
        t.nparts = partial0;
    } else {
        t.nparts = (int)t.nchunks;     // sum of squares and chunk maxima recomputed from the series
        if ((n = launch_trigger_reduce(t, st)) < 0) return LOFAR_E_CUDA;
        p->launches += n;
    }
    if ((n = launch_trigger_sigma(t, st)) < 0) return LOFAR_E_CUDA;
    p->launches += n;
    if (!emit) {
        if ((n = launch_trigger_flag(t, st)) < 0) return LOFAR_E_CUDA;
        p->launches += n;
        if (rescan) {
            RescanArgs r{};
            r.X = X; r.xpitch = T; r.dtype = p->dtype; r.T = T;
            r.W = p->dW; r.Dph = p->dDph; r.S = p->S; r.K = p->K; r.k0 = p->k0; r.B = p->B; r.D = p->D;
            r.hist0 = p->dHist0; r.gs = p->dGs; r.tw = p->dTw;
            r.items = p->dItems; r.nitems = p->dNItems; r.items_cap = p->items_cap;
            r.sigma = sigma; r.kappa = (float)p->kappa;
            r.chunkmax = p->dChunkMax; r.chunkmax_pitch = p->chunkmax_pitch;
            r.cand = cand; r.count = count; r.cap = p->max_cand; r.offset = p->offset;
            if ((n = launch_rescan(r, p->num_sms, st)) < 0) return LOFAR_E_CUDA;
        } else {
            if ((n = launch_trigger_scan(t, 4 * p->num_sms, st)) < 0) return LOFAR_E_CUDA;
        }
        p->launches += n;
    }
    if ((n = launch_trigger_sort(t, (emit || rescan) && p->D > 1, st)) < 0) return LOFAR_E_CUDA;
    p->launches += n;
    if (p->env_window > 1) {
        if ((n = launch_tail_save(series, N, N, ns, p->env_window, p->dTail, st)) < 0) return LOFAR_E_CUDA;
        p->launches += n;
    }
    if (causal) {
        // this block's sigma is the level the next block is measured against
        if ((n = launch_sigma_ref(sigma, (float)p->kappa, ns, p->dSigmaRef, p->dThr, st)) < 0) return LOFAR_E_CUDA;
        p->launches += n;
        p->have_ref = true;
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
    free_tables(p);                    // drains the plan's own streams first
    if (p->s_copy) { cudaStreamDestroy(p->s_copy); p->s_copy = nullptr; }
    if (p->s_comp) { cudaStreamDestroy(p->s_comp); p->s_comp = nullptr; }
    if (p->s_bf) { cudaStreamDestroy(p->s_bf); p->s_bf = nullptr; }
    if (p->s_ippf) { cudaStreamDestroy(p->s_ippf); p->s_ippf = nullptr; }
    if (p->ev_fork) cudaEventDestroy(p->ev_fork);
    if (p->ev_join) cudaEventDestroy(p->ev_join);
    for (int i = 0; i < 2; ++i) {
        if (p->ev_copied[i]) cudaEventDestroy(p->ev_copied[i]);
        if (p->ev_done[i]) cudaEventDestroy(p->ev_done[i]);
        if (p->ev_bf[i]) cudaEventDestroy(p->ev_bf[i]);
        if (p->ev_ippf[i]) cudaEventDestroy(p->ev_ippf[i]);
    }
    if (p->hCount) cudaFreeHost(p->hCount);
    for (auto &r : p->prof_pending) { cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
    for (auto e : p->prof_pool) cudaEventDestroy(e);
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
    const Layout L = layout(p);
    *bytes = L.table_bytes() + L.staging_bytes();
    return LOFAR_OK;
}

lofar_status lofar_plan_set_allocator(lofar_plan *p, void *(*alloc)(size_t, void *), void (*free_)(void *, void *),
                                      void *ctx)
{
    if (!p || ((alloc == nullptr) != (free_ == nullptr))) return LOFAR_E_INVALID;
    free_tables(p);                    // with the allocator that made them
    p->alloc_fn = alloc; p->free_fn = free_; p->alloc_ctx = ctx;
    return LOFAR_OK;
}

lofar_status lofar_plan_set_dedispersion(lofar_plan *p, lofar_dedispersion mode)
{
    if (!p || (mode != LOFAR_DEDISP_SUBBAND && mode != LOFAR_DEDISP_EXACT)) return LOFAR_E_INVALID;
    p->dedisp = mode;
    p->built = false;
    return LOFAR_OK;
}

lofar_status lofar_plan_set_inversion(lofar_plan *p, lofar_inversion mode, int iterations)
{
    if (!p || (mode != LOFAR_INV_MATCHED && mode != LOFAR_INV_LSMR)) return LOFAR_E_INVALID;
    if (mode == LOFAR_INV_LSMR && iterations <= 0) return LOFAR_E_INVALID;
    p->inversion = mode;
    if (mode == LOFAR_INV_LSMR) p->lsmr_iters = iterations;
    p->built = false;
    return LOFAR_OK;
}

lofar_status lofar_plan_set_sigma_mode(lofar_plan *p, lofar_sigma_mode mode, const float *sigma_init)
{
    if (!p || (mode != LOFAR_SIGMA_BLOCK && mode != LOFAR_SIGMA_CAUSAL)) return LOFAR_E_INVALID;
    p->sigma_mode = mode;
    if (sigma_init && mode == LOFAR_SIGMA_CAUSAL) p->sigma_init.assign(sigma_init, sigma_init + (size_t)p->B * p->D);
    else p->sigma_init.clear();
    p->built = false;
    return LOFAR_OK;
}

lofar_status lofar_cluster(lofar_plan *p, const lofar_candidate *cand, const uint32_t *count, uint64_t gap,
                           lofar_event *events, uint32_t *nevents, uint32_t max_events, void *stream)
{
    if (!p || !cand || !count || !events || !nevents || max_events == 0) return LOFAR_E_INVALID;
    const int n = launch_cluster(cand, count, p->max_cand, p->D, gap, events, nevents, max_events,
                                 static_cast<cudaStream_t>(stream));
    if (n < 0) return LOFAR_E_CUDA;
    p->launches += n;
    return LOFAR_OK;
}

lofar_status lofar_plan_set_scratch_limit(lofar_plan *p, size_t bytes)
{
    if (!p || bytes == 0) return LOFAR_E_INVALID;
    p->scratch_limit = bytes;
    p->built = false;
    return LOFAR_OK;
}

lofar_status lofar_plan_set_overlap(lofar_plan *p, int mode, int chunk_slices)
{
    if (!p || (mode != 0 && mode != 1) || chunk_slices < 0) return LOFAR_E_INVALID;
    p->overlap = mode;
    p->overlap_chunk = chunk_slices > 0 ? chunk_slices : 8192;
    p->built = false;
    return LOFAR_OK;
}

lofar_status lofar_plan_chunk_info(lofar_plan *p, int slices, int chunk, int64_t *first_slice, int64_t *chunk_slices,
                                   int *spans, int *span_slices)
{
    if (!p || slices <= 0 || chunk < 0 || !first_slice || !chunk_slices || !spans || !span_slices) return LOFAR_E_INVALID;
    if (p->max_slices > 0 && slices > p->max_slices) return LOFAR_E_STATE;
    const int keep = p->max_slices;
    if (p->max_slices <= 0) p->max_slices = slices;
    const Layout L = layout(p);
    p->max_slices = keep;
    int sms = p->num_sms;
    if (!p->built) {
        int dev = 0;
        if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        else { cudaGetLastError(); sms = 148; }
    }
    const long long c0 = (long long)chunk * L.zchunk;
    *first_slice = c0; *chunk_slices = 0; *spans = 0; *span_slices = 0;
    if (c0 >= slices) return LOFAR_OK;                       // past the last chunk
    const long long nc = slices - c0 < L.zchunk ? slices - c0 : L.zchunk;
    const bool lanes = L.overlap && slices > L.zchunk;
    *chunk_slices = nc;
    plan_spans((nc + kStepSlices - 1) / kStepSlices, p->ninv(), ippf_sm_budget(sms, lanes), lanes, spans, span_slices);
    return LOFAR_OK;
}

lofar_status lofar_plan_chunking(lofar_plan *p, int slices, int64_t *chunk_slices, int *spans, int *span_slices)
{
    int64_t first = 0;
    return lofar_plan_chunk_info(p, slices, 0, &first, chunk_slices, spans, span_slices);
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

lofar_status lofar_requantize(lofar_plan *p, const void *Z, int slices, float scale, void *X2, void *stream)
{
    if (!p || !Z || !X2 || slices <= 0 || !(scale > 0.f)) return LOFAR_E_INVALID;
    if ((reinterpret_cast<size_t>(Z) & 7) || (reinterpret_cast<size_t>(X2) & 15)) return LOFAR_E_ALIGN;
    const int n = launch_requantize(static_cast<const float2 *>(Z), (long long)p->K * slices, p->B * p->D, scale, X2,
                                    static_cast<cudaStream_t>(stream));
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
    if ((s = apply_reset(p, static_cast<cudaStream_t>(stream))) != LOFAR_OK) return s;
    int partial0 = 0;
    if (p->inversion == LOFAR_INV_LSMR) {
        cudaStream_t st = static_cast<cudaStream_t>(stream);
        if ((s = lsmr_begin(p, st)) != LOFAR_OK) return s;
        if ((s = do_ippf(p, static_cast<const float2 *>(Z), slices, 0, slices, 0, nullptr, (long long)slices * kMfft, 0,
                         &partial0, 0, st, EmitTo{nullptr, nullptr}, true)) != LOFAR_OK) return s;
        return lsmr_solve(p, slices, series, (long long)slices * kMfft, st);
    }
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
    if ((s = apply_reset(p, st)) != LOFAR_OK) return s;
    const long long N = (long long)slices * kMfft;
    const bool causal = p->sigma_mode == LOFAR_SIGMA_CAUSAL;
    if (causal && p->env_window != 1) return LOFAR_E_INVALID;
    TriggerArgs t = trigger_args(p, series, N, cand, count, sigma);
    t.nparts = (int)t.nchunks;
    int n;
    ProfScope prof(p, 2, st);
    if ((n = launch_trigger_reduce(t, st)) < 0) return LOFAR_E_CUDA;
    p->launches += n;
    if ((n = launch_trigger_sigma(t, st)) < 0) return LOFAR_E_CUDA;
    p->launches += n;
    if ((n = launch_trigger_flag(t, st)) < 0) return LOFAR_E_CUDA;
    p->launches += n;
    if ((n = launch_trigger_scan(t, 4 * p->num_sms, st)) < 0) return LOFAR_E_CUDA;
    p->launches += n;
    if ((n = launch_trigger_sort(t, false, st)) < 0) return LOFAR_E_CUDA;
    p->launches += n;
    if (p->env_window > 1) {
        if ((n = launch_tail_save(series, N, N, p->B * p->D, p->env_window, p->dTail, st)) < 0) return LOFAR_E_CUDA;
        p->launches += n;
    }
    if (causal) {
        if ((n = launch_sigma_ref(sigma, (float)p->kappa, p->B * p->D, p->dSigmaRef, p->dThr, st)) < 0) return LOFAR_E_CUDA;
        p->launches += n;
        p->have_ref = true;
    }
    p->offset += (uint64_t)N;
    return LOFAR_OK;
}

lofar_status lofar_run_block(lofar_plan *p, const void *X, int slices, float *series, lofar_candidate *cand,
                             uint32_t *count, float *sigma, void *stream)
{
    lofar_status s = ensure(p, slices);
    if (s != LOFAR_OK) return s;
    if (!cand || !count || !sigma) return LOFAR_E_INVALID;      // series == NULL: trigger-only
    if ((s = check_x(p, X, slices)) != LOFAR_OK) return s;
    if ((s = apply_reset(p, static_cast<cudaStream_t>(stream))) != LOFAR_OK) return s;
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
    p->reset_pending = p->built;       // zeroing is enqueued on the stream of the next compute call
    return LOFAR_OK;
}

lofar_status lofar_stream_push(lofar_plan *p, const void *X_host, int slices, float *series,
                               lofar_candidate *cand_host, uint32_t *count_host, float *sigma_host)
{
    lofar_status s = ensure(p, slices);
    if (s != LOFAR_OK) return s;
    if (!X_host) return LOFAR_E_INVALID;                        // series == NULL: trigger-only
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
        const Layout L = layout(p);
        for (int i = 0; i < 2 && s == LOFAR_OK; ++i) {
            char *x = nullptr;
            if ((s = dev_alloc(p, &x, L.x_bytes)) == LOFAR_OK) p->dX[i] = x;
            if (s == LOFAR_OK) s = dev_alloc(p, &p->dCand[i], L.cand);
            if (s == LOFAR_OK) s = dev_alloc(p, &p->dCount[i], 1);
            if (s == LOFAR_OK) s = dev_alloc(p, &p->dSigma[i], L.sigma);
        }
        if (s != LOFAR_OK) { free_staging(p); return s; }   // nothing half-allocated is left behind
        p->dX_bytes = L.x_bytes;
    }
    const int slot = (int)(p->push_index & 1);
    const size_t bytes = (size_t)p->S * 2 * p->K * (size_t)slices * sample_bytes(p);
    if (p->slot_used[slot]) CU(cudaStreamWaitEvent(p->s_copy, p->ev_done[slot], 0));
    CU(cudaMemcpyAsync(p->dX[slot], X_host, bytes, cudaMemcpyHostToDevice, p->s_copy));
    CU(cudaEventRecord(p->ev_copied[slot], p->s_copy));
    CU(cudaStreamWaitEvent(p->s_comp, p->ev_copied[slot], 0));
    if ((s = apply_reset(p, p->s_comp)) != LOFAR_OK) return s;
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

// ---- carried state for checkpoint / resume: header, history, envelope tail ----
namespace {
struct StateHeader { uint32_t magic, nseries, taps, fft, env_window, reserved; uint64_t offset; };
constexpr uint32_t kStateMagic = 0x4c4f4631u;   // "LOF1"
size_t state_bytes(const lofar_plan *p)
{
    const size_t ns = (size_t)p->B * p->D, ni = (size_t)p->ninv();
    const size_t xt = p->dedisp == LOFAR_DEDISP_EXACT ? (size_t)p->B * 2 * kMfft : 0;   // exact de-dispersion: two slices per beam
    return sizeof(StateHeader) + ni * (kTaps - 1) * kMfft * sizeof(float) + ns * (size_t)(p->env_window - 1) * sizeof(float) +
           ns * sizeof(float) +                // the causal reference level (header.reserved = 1 if valid)
           xt * sizeof(float);
}
}  // namespace

lofar_status lofar_stream_state_bytes(lofar_plan *p, size_t *bytes)
{
    if (!p || !bytes) return LOFAR_E_INVALID;
    *bytes = state_bytes(p);
    return LOFAR_OK;
}

lofar_status lofar_stream_get_state(lofar_plan *p, void *state_host, size_t bytes)
{
    if (!p || !state_host) return LOFAR_E_INVALID;
    if (bytes < state_bytes(p)) return LOFAR_E_SHAPE;
    if (!p->built) {
        if (p->max_slices <= 0) return LOFAR_E_STATE;
        const lofar_status st = build(p);
        if (st != LOFAR_OK) { free_tables(p); return st; }
    }
    quiesce(p);
    const size_t ns = (size_t)p->B * p->D, hist = (size_t)p->ninv() * (kTaps - 1) * kMfft * sizeof(float);
    const size_t tail = ns * (size_t)(p->env_window - 1) * sizeof(float);
    const size_t xt = p->dXhat ? (size_t)2 * kMfft * sizeof(float) : 0;
    StateHeader h{kStateMagic, (uint32_t)ns, (uint32_t)kTaps, (uint32_t)kMfft, (uint32_t)p->env_window,
                  (p->have_ref && !p->reset_pending) ? 1u : 0u, p->offset};
    char *dst = static_cast<char *>(state_host);
    std::memcpy(dst, &h, sizeof(h));
    std::memset(dst + sizeof(h), 0, hist + tail + ns * sizeof(float) + xt * p->B);
    if (p->reset_pending) return LOFAR_OK;
    if (xt) CU(cudaMemcpy2D(dst + sizeof(h) + hist + tail + ns * sizeof(float), xt, p->dXhat,
                            (size_t)p->xhat_pitch * sizeof(float), xt, (size_t)p->B, cudaMemcpyDeviceToHost));
    CU(cudaMemcpy(dst + sizeof(h), p->dHist[p->hist_parity], hist, cudaMemcpyDeviceToHost));
    if (tail) CU(cudaMemcpy(dst + sizeof(h) + hist, p->dTail, tail, cudaMemcpyDeviceToHost));
    if (h.reserved) CU(cudaMemcpy(dst + sizeof(h) + hist + tail, p->dSigmaRef, ns * sizeof(float), cudaMemcpyDeviceToHost));
    return LOFAR_OK;
}

lofar_status lofar_stream_set_state(lofar_plan *p, const void *state_host, size_t bytes)
{
    if (!p || !state_host) return LOFAR_E_INVALID;
    if (bytes < state_bytes(p)) return LOFAR_E_SHAPE;
    StateHeader h;
    std::memcpy(&h, state_host, sizeof(h));
    const size_t ns = (size_t)p->B * p->D;
    if (h.magic != kStateMagic || h.nseries != ns || h.taps != (uint32_t)kTaps || h.fft != (uint32_t)kMfft ||
        h.env_window != (uint32_t)p->env_window)
        return LOFAR_E_SHAPE;
    if (!p->built) {
        if (p->max_slices <= 0) return LOFAR_E_STATE;
        const lofar_status st = build(p);
        if (st != LOFAR_OK) { free_tables(p); return st; }
    }
    quiesce(p);
    const size_t hist = (size_t)p->ninv() * (kTaps - 1) * kMfft * sizeof(float), tail = ns * (size_t)(p->env_window - 1) * sizeof(float);
    const char *src = static_cast<const char *>(state_host);
    if (p->dXhat) {
        const size_t xt = (size_t)2 * kMfft * sizeof(float);
        CU(cudaMemcpy2D(p->dXhat, (size_t)p->xhat_pitch * sizeof(float), src + sizeof(h) + hist + tail + ns * sizeof(float), xt,
                        xt, (size_t)p->B, cudaMemcpyHostToDevice));
    }
    CU(cudaMemcpy(p->dHist[p->hist_parity], src + sizeof(h), hist, cudaMemcpyHostToDevice));
    if (tail) CU(cudaMemcpy(p->dTail, src + sizeof(h) + hist, tail, cudaMemcpyHostToDevice));
    p->have_ref = false;
    if (h.reserved && p->sigma_mode == LOFAR_SIGMA_CAUSAL) {
        std::vector<float> ref(ns), thr(ns);
        std::memcpy(ref.data(), src + sizeof(h) + hist + tail, ns * sizeof(float));
        for (size_t i = 0; i < ns; ++i) thr[i] = (float)p->kappa * ref[i];
        CU(cudaMemcpy(p->dSigmaRef, ref.data(), ns * sizeof(float), cudaMemcpyHostToDevice));
        CU(cudaMemcpy(p->dThr, thr.data(), ns * sizeof(float), cudaMemcpyHostToDevice));
        p->have_ref = true;
    }
    p->offset = h.offset;
    p->reset_pending = false;
    return LOFAR_OK;
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
        if (r.id >= 0 && r.id < LOFAR_PROFILE_SLOTS) { ms[r.id] += (double)t; launches[r.id] += 1; }
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
