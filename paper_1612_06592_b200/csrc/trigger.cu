// trigger.cu -- step a5: amplitude threshold trigger ("Triggering on the amplitude of a
// pulse"; definitions O7/O8 and readings A13-A15 in DESIGN.md).
//
//   e[n]     = sqrt( (1/W) sum_{j<W} xhat[n-j]^2 )                 (W = 1: e = |xhat|)
//   sigma[s] = sqrt( (1/N) sum_n e[n]^2 ) over this block
//   D = 1: candidate iff e/sigma > kappa.   D > 1: per (beam, n) the trial with the largest
//   e/sigma (lowest d on ties) is the candidate iff that ratio > kappa.
//
// sum e^2 and the per-16384-sample maximum of e normally come out of the inverse-PPF epilogue
// (ippf.cu); the reduce kernel here recomputes them from a series in HBM for the stand-alone stage
// call and for W > 1.  A flag kernel lists the 16384-sample chunks whose maximum can reach the threshold;
// the scan kernel re-reads the series only there (or, without a series, ippf.cu's rescan kernel recomputes
// them); survivors are compacted with a warp ballot and one atomic per warp, sorted by (beam, sample) by a
// single CTA and reduced to the best trial per sample.  With a causal sigma (threshold known before the
// block) the candidates come straight out of the inverse-PPF epilogue and only the sort runs here.
// cluster_kernel groups the sorted list into events.
#include "plan.h"

namespace lofar {
namespace {

constexpr int kChunk = 16384;   // samples per pruning chunk = 16 slices

__device__ __forceinline__ float env_sq(const float *x, const float *tail, long long n, int W)
{
    // (1/W) * sum_{j<W} x[n-j]^2 with x[-1..-(W-1)] taken from tail[W-2 .. 0]
    float s = 0.f;
    for (int j = 0; j < W; ++j) {
        const long long i = n - j;
        const float v = (i >= 0) ? x[i] : tail[(W - 1) + i];
        s = fmaf(v, v, s);
    }
    return s / (float)W;
}

__global__ void __launch_bounds__(256) reduce_kernel(TriggerArgs a)
{
    const int series = blockIdx.y;
    const long long c = blockIdx.x;
    const float *x = a.series + (size_t)series * a.series_pitch;
    const float *tail = a.tail ? a.tail + (size_t)series * (a.W - 1) : nullptr;
    const long long n0 = c * kChunk;
    const long long n1 = (n0 + kChunk < a.N) ? n0 + kChunk : a.N;
    float s = 0.f, m = 0.f;
    for (long long n = n0 + threadIdx.x; n < n1; n += 256) {
        const float e2 = (a.W == 1) ? x[n] * x[n] : env_sq(x, tail, n, a.W);
        s += e2;
        m = fmaxf(m, e2);
    }
    double ds = (double)s;
    __shared__ double sd[8];
    __shared__ float sm[8];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        ds += __shfl_xor_sync(0xffffffffu, ds, o);
        m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
    }
    if ((threadIdx.x & 31) == 0) { sd[threadIdx.x >> 5] = ds; sm[threadIdx.x >> 5] = m; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0; float mm = 0.f;
        for (int w = 0; w < 8; ++w) { t += sd[w]; mm = fmaxf(mm, sm[w]); }
        a.partial[(size_t)series * a.partial_pitch + c] = t;
        a.chunkmax[(size_t)series * a.chunkmax_pitch + c] = sqrtf(mm);
    }
}

__global__ void __launch_bounds__(256) sigma_kernel(TriggerArgs a)
{
    const int series = blockIdx.x;
    const double *p = a.partial + (size_t)series * a.partial_pitch;
    double s = 0.0;
    for (int i = threadIdx.x; i < a.nparts; i += 256) s += p[i];
    __shared__ double sd[8];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) sd[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int w = 0; w < 8; ++w) t += sd[w];
        a.sigma[series] = (float)sqrt(t / (double)a.N);
        if (series == 0) {
            if (a.zero_count) *a.count = 0u;
            *a.nitems = 0u;
        }
    }
}

// One thread per (beam, chunk): can any trial of this beam reach its threshold inside this chunk?
__global__ void __launch_bounds__(256) flag_kernel(TriggerArgs a)
{
    const long long c = (long long)blockIdx.x * 256 + threadIdx.x;
    const int b = blockIdx.y;
    if (c >= a.nchunks) return;
    bool any = false;
    for (int d = 0; d < a.D; ++d) {
        const int s = b * a.D + d;
        const float cm = a.chunkmax[(size_t)s * a.chunkmax_pitch + c];
        if (cm >= a.kappa * a.sigma_thr[s] * 0.99999f) any = true;
    }
    if (any) {
        const uint32_t slot = atomicAdd(a.nitems, 1u);
        if (slot < a.items_cap) a.items[slot] = make_int2(b, (int)c);
    }
}

// Threshold scan of the flagged chunks (the series is re-read only there); survivors are compacted with a warp
// ballot and one atomic per warp.  If the list overflowed (a threshold far inside the noise) every chunk is scanned.
__global__ void __launch_bounds__(256) scan_kernel(TriggerArgs a)
{
    const int D = a.D;
    const uint32_t listed = *a.nitems;
    const bool all = listed > a.items_cap;
    const long long total = all ? a.nchunks * a.B : (long long)listed;
    const int lane = threadIdx.x & 31;
    for (long long it = blockIdx.x; it < total; it += gridDim.x) {
        const int b = all ? (int)(it / a.nchunks) : a.items[it].x;
        const long long c = all ? it % a.nchunks : a.items[it].y;
        const long long n0 = c * kChunk;
        const long long n1 = (n0 + kChunk < a.N) ? n0 + kChunk : a.N;
        if (a.W == 1 && D == 1) {
            // one series per beam, envelope = |x|: four rows of 256 samples are loaded before any is judged (when the
            // flag list overflowed the whole series streams through here)
            const float *x = a.series + (size_t)b * a.series_pitch;
            const float sig = a.sigma_thr[b];
            for (long long nb = n0; nb < n1; nb += 1024) {
                float ev[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const long long n = nb + u * 256 + threadIdx.x;
                    ev[u] = n < n1 ? fabsf(x[n]) : -1.f;
                }
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const long long n = nb + u * 256 + threadIdx.x;
                    const bool hit = ev[u] >= 0.f && ev[u] / sig > a.kappa;
                    const unsigned mask = __ballot_sync(0xffffffffu, hit);
                    if (mask) {
                        unsigned base = 0;
                        if (lane == 0) base = atomicAdd(a.count, (unsigned)__popc(mask));
                        base = __shfl_sync(0xffffffffu, base, 0);
                        if (hit) {
                            const unsigned slot = base + __popc(mask & ((1u << lane) - 1u));
                            if (slot < a.cap) {
                                lofar_candidate r;
                                r.series = (uint32_t)b; r.trial = 0u;
                                r.sample = a.offset + (uint64_t)n;
                                r.env = ev[u]; r.sigma = sig;
                                a.cand[slot] = r;
                            }
                        }
                    }
                }
            }
            continue;
        }
        for (long long nb = n0; nb < n1; nb += 256) {
            const long long n = nb + threadIdx.x;
            bool hit = false;
            int best = 0;
            float best_e = 0.f, best_snr = -1.f;
            if (n < n1) {
                for (int d = 0; d < D; ++d) {
                    const int s = b * D + d;
                    const float *x = a.series + (size_t)s * a.series_pitch;
                    float e;
                    if (a.W == 1) e = fabsf(x[n]);
                    else e = sqrtf(env_sq(x, a.tail + (size_t)s * (a.W - 1), n, a.W));
                    const float snr = e / a.sigma_thr[s];
                    if (snr > best_snr) { best_snr = snr; best = d; best_e = e; }
                }
                hit = best_snr > a.kappa;
            }
            const unsigned mask = __ballot_sync(0xffffffffu, hit);
            if (mask) {
                unsigned base = 0;
                if (lane == 0) base = atomicAdd(a.count, (unsigned)__popc(mask));
                base = __shfl_sync(0xffffffffu, base, 0);
                if (hit) {
                    const unsigned slot = base + __popc(mask & ((1u << lane) - 1u));
                    if (slot < a.cap) {
                        lofar_candidate r;
                        r.series = (uint32_t)(b * D + best);
                        r.trial = (uint32_t)best;
                        r.sample = a.offset + (uint64_t)n;
                        r.env = best_e;
                        r.sigma = a.sigma_thr[b * D + best];
                        a.cand[slot] = r;
                    }
                }
            }
        }
    }
}

// Order: beam, sample, then (for records of several trials at one sample) larger e/sigma first, lower trial first.
__device__ __forceinline__ bool cand_after(const lofar_candidate &x, const lofar_candidate &y, int D)
{
    const uint32_t bx = x.series / D, by = y.series / D;
    if (bx != by) return bx > by;
    if (x.sample != y.sample) return x.sample > y.sample;
    const float sx = x.env / x.sigma, sy = y.env / y.sigma;
    if (sx != sy) return sx < sy;
    return x.trial > y.trial;
}

// Direction-free bitonic network (every compare-exchange puts the smaller key first), so the
// virtual +inf padding beyond n never has to move.  One CTA; records live in global memory.
__global__ void __launch_bounds__(1024) sort_kernel(TriggerArgs a)
{
    const uint32_t total = *a.count;
    const uint32_t n = total < a.cap ? total : a.cap;
    if (n < 2) return;
    uint32_t n2 = 1;
    while (n2 < n) n2 <<= 1;
    for (uint32_t k = 2; k <= n2; k <<= 1) {
        for (uint32_t j = k >> 1; j > 0; j >>= 1) {
            const bool flip = (j == (k >> 1));
            for (uint32_t i = threadIdx.x; i < n; i += 1024) {
                const uint32_t l = flip ? (i ^ (k - 1)) : (i ^ j);
                if (l > i && l < n) {
                    lofar_candidate x = a.cand[i], y = a.cand[l];
                    if (cand_after(x, y, a.D)) { a.cand[i] = y; a.cand[l] = x; }
                }
            }
            __syncthreads();
        }
    }
}

// Best trial per (beam, sample): of equal keys the sorted list keeps the first record (largest e/sigma, lowest
// trial on ties; reading A15).  In-place compaction by one CTA in rounds of 1024 records; *count becomes the number
// of distinct candidates (left as the raw total if the buffer overflowed: the caller sees the overflow).
__global__ void __launch_bounds__(1024) unique_kernel(TriggerArgs a)
{
    __shared__ uint32_t swarp[32];
    __shared__ uint32_t sbase;
    __shared__ uint32_t prev_beam;
    __shared__ unsigned long long prev_sample;
    const uint32_t total = *a.count;
    if (total > a.cap || total < 2) return;
    const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
    if (t == 0) { sbase = 0; prev_beam = 0xffffffffu; prev_sample = 0ull; }
    __syncthreads();
    for (uint32_t r0 = 0; r0 < total; r0 += 1024) {
        const uint32_t i = r0 + t;
        lofar_candidate me;
        bool keep = false;
        if (i < total) {
            me = a.cand[i];
            uint32_t pb; unsigned long long ps;
            if (t == 0) { pb = prev_beam; ps = prev_sample; }
            else { const lofar_candidate p = a.cand[i - 1]; pb = p.series / a.D; ps = p.sample; }
            keep = (me.series / a.D != pb) || (me.sample != ps);
        }
        const unsigned m = __ballot_sync(0xffffffffu, keep);
        if (lane == 0) swarp[warp] = __popc(m);
        __syncthreads();                                  // every record of the round has been read
        uint32_t off = sbase;
        for (int w = 0; w < warp; ++w) off += swarp[w];
        if (keep) a.cand[off + __popc(m & ((1u << lane) - 1u))] = me;
        __syncthreads();
        if (t == 1023 || i == total - 1) {
            if (i < total) { prev_beam = me.series / a.D; prev_sample = me.sample; }
        }
        if (t == 0) { uint32_t s = 0; for (int w = 0; w < 32; ++w) s += swarp[w]; sbase += s; }
        __syncthreads();
    }
    if (t == 0) *a.count = sbase;
}

__global__ void sigma_ref_kernel(const float *sigma, float kappa, int nseries, float *sigma_ref, float *thr)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < nseries) { sigma_ref[i] = sigma[i]; thr[i] = kappa * sigma[i]; }
}

// Time clustering of one block's sorted candidate list into events (reading A22): consecutive
// candidates of a beam whose samples differ by at most `gap` form an event; its peak is the candidate with the
// largest e/sigma (lowest sample on ties).  One CTA: every thread owns a contiguous piece of the list, counts the
// events that start in it, and after a scan of those counts walks each of its events to the end.
__global__ void __launch_bounds__(1024) cluster_kernel(const lofar_candidate *cand, const uint32_t *count, uint32_t cap,
                                                       int D, unsigned long long gap, lofar_event *events,
                                                       uint32_t *nevents, uint32_t max_events)
{
    __shared__ uint32_t sscan[1024];
    const uint32_t total = *count < cap ? *count : cap;
    const uint32_t per = (total + 1023) / 1024;
    const uint32_t lo = min(threadIdx.x * per, total), hi = min(lo + per, total);
    auto starts = [&](uint32_t i) {
        if (i == 0) return true;
        const lofar_candidate p = cand[i - 1], c = cand[i];
        return (p.series / D != c.series / D) || (c.sample - p.sample > gap);
    };
    uint32_t mine = 0;
    for (uint32_t i = lo; i < hi; ++i) mine += starts(i) ? 1u : 0u;
    sscan[threadIdx.x] = mine;
    __syncthreads();
    for (int o = 1; o < 1024; o <<= 1) {
        const uint32_t v = threadIdx.x >= o ? sscan[threadIdx.x - o] : 0u;
        __syncthreads();
        sscan[threadIdx.x] += v;
        __syncthreads();
    }
    uint32_t slot = sscan[threadIdx.x] - mine;
    if (threadIdx.x == 1023) *nevents = sscan[1023];
    for (uint32_t i = lo; i < hi; ++i) {
        if (!starts(i)) continue;
        uint32_t j = i, peak = i;
        float best = cand[i].env / cand[i].sigma;
        while (j + 1 < total && !starts(j + 1)) {
            ++j;
            const float s = cand[j].env / cand[j].sigma;
            if (s > best) { best = s; peak = j; }
        }
        if (slot < max_events) {
            lofar_event e;
            const lofar_candidate pk = cand[peak];
            e.beam = pk.series / D; e.count = j - i + 1;
            e.first_sample = cand[i].sample; e.last_sample = cand[j].sample; e.peak_sample = pk.sample;
            e.peak_trial = pk.trial; e.peak_env = pk.env; e.peak_sigma = pk.sigma; e.peak_snr = best;
            events[slot] = e;
        }
        ++slot;
    }
}

__global__ void tail_kernel(const float *series, long long pitch, long long N, int nseries, int W, float *tail)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int n = nseries * (W - 1);
    if (i >= n) return;
    const int s = i / (W - 1), j = i - s * (W - 1);
    tail[i] = series[(size_t)s * pitch + (N - (W - 1) + j)];
}

}  // namespace

int launch_trigger_reduce(const TriggerArgs &a, cudaStream_t st)
{
    dim3 grid((unsigned)a.nchunks, (unsigned)(a.B * a.D));
    reduce_kernel<<<grid, 256, 0, st>>>(a);
    return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

int launch_trigger_sigma(const TriggerArgs &a, cudaStream_t st)
{
    sigma_kernel<<<a.B * a.D, 256, 0, st>>>(a);
    return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

int launch_trigger_flag(const TriggerArgs &a, cudaStream_t st)
{
    dim3 grid((unsigned)((a.nchunks + 255) / 256), (unsigned)a.B);
    flag_kernel<<<grid, 256, 0, st>>>(a);
    return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

int launch_trigger_scan(const TriggerArgs &a, int grid, cudaStream_t st)
{
    scan_kernel<<<grid, 256, 0, st>>>(a);
    return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

int launch_trigger_sort(const TriggerArgs &a, bool unique, cudaStream_t st)
{
    sort_kernel<<<1, 1024, 0, st>>>(a);
    if (unique) unique_kernel<<<1, 1024, 0, st>>>(a);
    return cudaGetLastError() == cudaSuccess ? (unique ? 2 : 1) : -1;
}

int launch_sigma_ref(const float *sigma, float kappa, int nseries, float *sigma_ref, float *thr, cudaStream_t st)
{
    sigma_ref_kernel<<<(nseries + 255) / 256, 256, 0, st>>>(sigma, kappa, nseries, sigma_ref, thr);
    return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

int launch_cluster(const lofar_candidate *cand, const uint32_t *count, uint32_t cap, int D, uint64_t gap,
                   lofar_event *events, uint32_t *nevents, uint32_t max_events, cudaStream_t st)
{
    cluster_kernel<<<1, 1024, 0, st>>>(cand, count, cap, D, (unsigned long long)gap, events, nevents, max_events);
    return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

int launch_tail_save(const float *series, long long pitch, long long N, int nseries, int W, float *tail,
                     cudaStream_t st)
{
    const int n = nseries * (W - 1);
    if (n <= 0) return 0;
    tail_kernel<<<(n + 255) / 256, 256, 0, st>>>(series, pitch, N, nseries, W, tail);
    return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

}  // namespace lofar
