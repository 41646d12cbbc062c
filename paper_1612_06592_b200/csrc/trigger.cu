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
// call and for W > 1.  The scan kernel skips every 16384-sample chunk whose maximum cannot reach the
// threshold, so the series is re-read only around pulses; survivors are compacted with a warp ballot
// and one atomic per warp, then sorted by (beam, sample) by a single CTA.
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
        if (series == 0) *a.count = 0u;
    }
}

__global__ void __launch_bounds__(256) scan_kernel(TriggerArgs a)
{
    const int b = blockIdx.y;
    const long long c = blockIdx.x;
    const int D = a.D;
    // prune: can any trial of this beam reach the threshold inside this chunk?
    bool any = false;
    for (int d = 0; d < D; ++d) {
        const int s = b * D + d;
        const float cm = a.chunkmax[(size_t)s * a.chunkmax_pitch + c];
        if (cm >= a.kappa * a.sigma[s] * 0.99999f) any = true;
    }
    if (!any) return;

    const long long n0 = c * kChunk;
    const long long n1 = (n0 + kChunk < a.N) ? n0 + kChunk : a.N;
    const int lane = threadIdx.x & 31;
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
                const float snr = e / a.sigma[s];
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
                    r.sigma = a.sigma[b * D + best];
                    a.cand[slot] = r;
                }
            }
        }
    }
}

__device__ __forceinline__ bool cand_after(const lofar_candidate &x, const lofar_candidate &y, int D)
{
    const uint32_t bx = x.series / D, by = y.series / D;
    return bx > by || (bx == by && x.sample > y.sample);
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

int launch_trigger_finish(const TriggerArgs &a, cudaStream_t st)
{
    sigma_kernel<<<a.B * a.D, 256, 0, st>>>(a);
    dim3 grid((unsigned)a.nchunks, (unsigned)a.B);
    scan_kernel<<<grid, 256, 0, st>>>(a);
    sort_kernel<<<1, 1024, 0, st>>>(a);
    return cudaGetLastError() == cudaSuccess ? 3 : -1;
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
