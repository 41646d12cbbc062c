// ippf.cu -- steps a3 + a4 (+ the sum of squares and per-step maximum that a5 needs):
// inversion of the polyphase filter bank (section 3: "an inverse Fourier
// transformation F^-1 y~ = y of the filtered signal" followed by the FIR system H; here one
// application of the matched synthesis FIR g = 1024 h, reading A8).
//
// One CTA (512 threads, 16 warps) owns one series and marches along a span of time slices in
// steps of 16 slices:
//   pre-pass : reads the K selected sub-band rows of Z for 16 slices (one 128-byte line per row),
//              applies the trial phasor if asked, builds the packed half-spectrum V (fft_math.cuh)
//              and stores it transposed -- slice-major -- into shared memory;
//   FFT      : warp w transforms slice w in place: a radix-16 and a radix-32 pass (fft512_warp);
//   FIR      : thread n owns output residues r = 2n, 2n+1; the 31-slice window (15 carried + 16 new)
//              is read from the previous and current slice buffers, the 16 taps from shared memory;
//              16 x 1024 contiguous output samples are written per step.
// The 15-slice history lives in the "previous" shared-memory buffer, is loaded from the plan at the
// start of a block and written back by the CTA that owns the last span; CTAs that start in the
// middle of a block first transform the 16 slices before their span (no output).
#include "fft_math.cuh"
#include "plan.h"

namespace lofar {
namespace {

constexpr int kThreads = 512;
constexpr int kTwCount = 256 + 512;        // w1024[256], TB[32][16] = exp(2 pi i j r / 512)
constexpr size_t kSmemBytes = (size_t)(2 * kStep * kRow + kP * kH + kTwCount) * sizeof(float2) + 256;

struct Ctx {
    const float2 *Zs;      // rows of this series' beam (sub-band j at Zs + j*zpitch)
    const float2 *ph;      // trial phasors of this series or nullptr
    long long zpitch, nc;
    int K, k0, vec_ok, tiled;
};

// Two consecutive slices (col, col+1) of absolute sub-band k; zero outside the selected band / launch.
__device__ __forceinline__ float4 load2(const Ctx &c, int k, long long col)
{
    const int j = k - c.k0;
    float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
    if (j < 0 || j >= c.K || col >= c.nc) return v;
    const float2 *p = c.tiled ? c.Zs + ((size_t)(col >> 5) * c.K + j) * 32 + (col & 31)
                              : c.Zs + (size_t)j * c.zpitch + col;
    if (col + 1 < c.nc) {
        if (c.vec_ok) {
            v = __ldcs(reinterpret_cast<const float4 *>(p));
        } else {
            float2 z0 = p[0], z1 = p[1];
            v = make_float4(z0.x, z0.y, z1.x, z1.y);
        }
    } else {
        float2 z0 = p[0];
        v.x = z0.x; v.y = z0.y;
    }
    return v;
}

// Global loads of one 16-slice step, held in registers so that they can be issued one step ahead:
// thread unit i covers conjugate pair m = (tid>>3) + 64 i (m = 0: bins 0 and 256) and slices 2tp, 2tp+1.
struct StepRegs { float4 a[4], b[4]; };

__device__ __forceinline__ void prefetch(const Ctx &c, long long q, int tid, StepRegs &r)
{
    const int tp = tid & 7, m0 = tid >> 3;
    const long long col = q + 2 * tp;
    if (c.vec_ok && col + 1 < c.nc) {
        // common case, branch-free: predicated 16-byte loads, rows outside the selected band read as zero
        // tiled scratch: 32-slice tiles [K][32]: a step reads 128 of every 256 bytes of one contiguous block; else rows zpitch apart
        const float2 *p0 = c.tiled ? c.Zs + (size_t)(col >> 5) * c.K * 32 + (col & 31) : c.Zs + col;
        const unsigned K = (unsigned)c.K, zp = c.tiled ? 32u : (unsigned)c.zpitch;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int m = m0 + 64 * i;
            const unsigned ja = (unsigned)(m - c.k0), jb = (unsigned)((m == 0 ? 256 : 512 - m) - c.k0);
            float4 va = make_float4(0.f, 0.f, 0.f, 0.f), vb = va;
            if (ja < K) va = __ldcs(reinterpret_cast<const float4 *>(p0 + (size_t)(ja * zp)));
            if (jb < K) vb = __ldcs(reinterpret_cast<const float4 *>(p0 + (size_t)(jb * zp)));
            r.a[i] = va; r.b[i] = vb;
        }
        // pull the rows of the step after this one into L2 (one 128-byte line per row: lanes with tp == 0)
        if (tp == 0 && col + 2 * kStep < c.nc) {
            const float2 *p1 = c.tiled ? c.Zs + (size_t)((col + kStep) >> 5) * c.K * 32 + ((col + kStep) & 31) : p0 + kStep;
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const int m = m0 + 64 * i;
                const unsigned ja = (unsigned)(m - c.k0), jb = (unsigned)((m == 0 ? 256 : 512 - m) - c.k0);
                if (ja < K) asm volatile("prefetch.global.L2 [%0];" :: "l"(p1 + (size_t)(ja * zp)));
                if (jb < K) asm volatile("prefetch.global.L2 [%0];" :: "l"(p1 + (size_t)(jb * zp)));
            }
        }
    } else {
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int m = m0 + 64 * i;
            r.a[i] = load2(c, m, col);
            r.b[i] = load2(c, m == 0 ? 256 : 512 - m, col);
        }
    }
}

// Pre-pass of the 16 slices held in r into dst[16][kRow] (packed half-spectrum V, slice-major).
__device__ __forceinline__ float4 rotate2(float4 v, float2 f)
{
    return make_float4(f.x * v.x - f.y * v.y, f.x * v.y + f.y * v.x, f.x * v.z - f.y * v.w, f.x * v.w + f.y * v.z);
}

__device__ __forceinline__ void prepass(const Ctx &c, const StepRegs &r, float2 *dst, const float2 *stw, int tid)
{
    const int tp = tid & 7, m0 = tid >> 3;
    float2 *r0 = dst + 2 * tp * kRow, *r1 = r0 + kRow;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const int m = m0 + 64 * i;
        float4 a = r.a[i], b = r.b[i];
        if (c.ph) {
            // STEC trial fan-out (a2): the trial's phasor multiplies the beam sums as they enter the transform
            const unsigned ja = (unsigned)(m - c.k0), jb = (unsigned)((m == 0 ? 256 : 512 - m) - c.k0);
            if (ja < (unsigned)c.K) a = rotate2(a, __ldg(c.ph + ja));
            if (jb < (unsigned)c.K) b = rotate2(b, __ldg(c.ph + jb));
        }
        if (m == 0) {
            r0[pad(0)] = prepass_dc(make_float2(a.x, a.y));
            r1[pad(0)] = prepass_dc(make_float2(a.z, a.w));
            r0[pad(256)] = prepass_quarter(make_float2(b.x, b.y));
            r1[pad(256)] = prepass_quarter(make_float2(b.z, b.w));
        } else {
            const float2 w = stw[m];
            float2 vm, vmir;
            prepass_pair(make_float2(a.x, a.y), make_float2(b.x, b.y), w, vm, vmir);
            r0[pad(m)] = vm; r0[pad(512 - m)] = vmir;
            prepass_pair(make_float2(a.z, a.w), make_float2(b.z, b.w), w, vm, vmir);
            r1[pad(m)] = vm; r1[pad(512 - m)] = vmir;
        }
    }
}

// 512-point inverse complex FFT of one slice row by one warp, in place: 512 = 16 x 32.
//   pass A: lane j does the 16-point DFT of elements j + 32 r and writes them to 16 j + m;
//   pass B: butterfly j (0..15) is a 32-point DFT of elements j + 16 r with twiddles exp(2 pi i j r / 512);
//           lanes j and j + 16 share it: each does the 16-point DFT of the even / odd r, the odd lane applies
//           W32^m, the halves are exchanged with shuffles; outputs go to j + 16 m (m < 16 low lane, m >= 16 high).
__device__ __forceinline__ void fft512_warp(float2 *row, const float2 *stw, int lane)
{
    float2 x[16];
#pragma unroll
    for (int r = 0; r < 16; ++r) x[r] = row[pad(lane + 32 * r)];
    idft16(x);
    __syncwarp();
#pragma unroll
    for (int m = 0; m < 16; ++m) row[pad(16 * lane + m)] = x[m];
    __syncwarp();
    const float2 *T = stw + 256 + lane;          // T[32 r' + lane] = exp(2 pi i j (hh + 2 r') / 512)
#pragma unroll
    for (int r = 0; r < 16; ++r) x[r] = cmul(row[pad(lane + 32 * r)], T[32 * r]);
    idft16(x);
    const bool hi = lane >= 16;
    if (hi) {
        // W32^m = exp(2 pi i m / 32), m = 0..15
        const float c[16] = {1.f, 0.98078528040323044913f, 0.92387953251128675613f, 0.83146961230254523708f,
                             0.70710678118654752440f, 0.55557023301960222474f, 0.38268343236508977173f,
                             0.19509032201612826785f, 0.f, -0.19509032201612826785f, -0.38268343236508977173f,
                             -0.55557023301960222474f, -0.70710678118654752440f, -0.83146961230254523708f,
                             -0.92387953251128675613f, -0.98078528040323044913f};
        const float sn[16] = {0.f, 0.19509032201612826785f, 0.38268343236508977173f, 0.55557023301960222474f,
                              0.70710678118654752440f, 0.83146961230254523708f, 0.92387953251128675613f,
                              0.98078528040323044913f, 1.f, 0.98078528040323044913f, 0.92387953251128675613f,
                              0.83146961230254523708f, 0.70710678118654752440f, 0.55557023301960222474f,
                              0.38268343236508977173f, 0.19509032201612826785f};
#pragma unroll
        for (int m = 1; m < 16; ++m) x[m] = cmul(x[m], make_float2(c[m], sn[m]));
    }
#pragma unroll
    for (int m = 0; m < 16; ++m) {
        float2 other;
        other.x = __shfl_xor_sync(0xffffffffu, x[m].x, 16);
        other.y = __shfl_xor_sync(0xffffffffu, x[m].y, 16);
        x[m] = hi ? csub(other, x[m]) : cadd(x[m], other);     // low lane: E + O', high lane: E - O'
    }
    __syncwarp();
    const int base = (lane & 15) + (hi ? 256 : 0);
#pragma unroll
    for (int m = 0; m < 16; ++m) row[pad(base + 16 * m)] = x[m];
    __syncwarp();
}

__global__ void __launch_bounds__(kThreads, 1) ippf_kernel(IppfArgs a)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2 *buf0 = reinterpret_cast<float2 *>(smem_raw);
    float2 *buf1 = buf0 + kStep * kRow;
    float2 *sg = buf1 + kStep * kRow;      // [16][512]
    float2 *stw = sg + kP * kH;            // [kTwCount]
    float *sred = reinterpret_cast<float *>(stw + kTwCount);   // 16 floats + 16 doubles (aligned)
    double *sdred = reinterpret_cast<double *>(sred + 32);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int series = blockIdx.x % a.nseries;
    const int span = blockIdx.x / a.nseries;
    const long long qs = (long long)span * a.span_len;
    if (qs >= a.nc) return;
    const long long qe = (qs + a.span_len < a.nc) ? qs + a.span_len : a.nc;
    const bool is_last = (qe == a.nc);

    Ctx c;
    const int zi = a.zmap_trials ? series / a.zmap_trials : series;
    c.Zs = a.Z + (size_t)zi * a.K * (size_t)a.zpitch;
    c.ph = a.zmap_trials ? a.Dph + (size_t)(series % a.zmap_trials) * a.K : nullptr;
    c.zpitch = a.zpitch; c.nc = a.nc; c.K = a.K; c.k0 = a.k0; c.vec_ok = a.vec_ok; c.tiled = a.ztile;

    for (int i = tid; i < kP * kH; i += kThreads) sg[i] = a.gs[i];
    for (int i = tid; i < kTwCount; i += kThreads) stw[i] = a.tw[i];

    float2 *prev = buf0, *cur = buf1;
    if (span == 0) {
        const float *h = a.hist_in + (size_t)series * (kP - 1) * kM;
#pragma unroll
        for (int i = 0; i < kP - 1; ++i)
            prev[(i + 1) * kRow + pad(tid)] = *reinterpret_cast<const float2 *>(h + (size_t)i * kM + 2 * tid);
        __syncthreads();
    } else {
        __syncthreads();   // twiddles visible
        StepRegs w;
        prefetch(c, qs - kStep, tid, w);
        prepass(c, w, cur, stw, tid);
        __syncthreads();
        fft512_warp(cur + warp * kRow, stw, lane);
        __syncthreads();
        float2 *t = prev; prev = cur; cur = t;
    }
    StepRegs regs;
    prefetch(c, qs, tid, regs);

    float *out = a.series ? a.series + (size_t)series * a.series_pitch + a.out0 : nullptr;
    double dsum = 0.0;

    for (long long q = qs; q < qe; q += kStep) {
        const int nvalid = (qe - q < kStep) ? (int)(qe - q) : kStep;
        prepass(c, regs, cur, stw, tid);
        if (q + kStep < qe) prefetch(c, q + kStep, tid, regs);   // next step's loads fly during FFT + FIR
        __syncthreads();
        fft512_warp(cur + warp * kRow, stw, lane);
        __syncthreads();

        // ---- synthesis FIR: out[j] = sum_t g[t] * win[15 + j - t] ----
        float2 g[kP], acc[kStep];
#pragma unroll
        for (int t = 0; t < kP; ++t) g[t] = sg[t * kH + tid];
#pragma unroll
        for (int j = 0; j < kStep; ++j) acc[j] = make_float2(0.f, 0.f);
        const int pn = pad(tid);
        float ssum = 0.f, smax = 0.f;
#pragma unroll
        for (int i = 0; i < kP - 1 + kStep; ++i) {
            const float2 x = (i < kP - 1) ? prev[(i + 1) * kRow + pn] : cur[(i - (kP - 1)) * kRow + pn];
#pragma unroll
            for (int t = 0; t < kP; ++t) {
                const int j = i - (kP - 1) + t;
                if (j >= 0 && j < kStep) {
                    acc[j].x = fmaf(g[t].x, x.x, acc[j].x);
                    acc[j].y = fmaf(g[t].y, x.y, acc[j].y);
                }
            }
            // output slice j = i - 15 is complete once window element i has been applied: store it now so
            // that the 64 KB of stores per step are spread over the second half of the FIR
            if (i >= kP - 1) {
                const int j = i - (kP - 1);
                if (j < nvalid) {
                    if (out) __stcs(reinterpret_cast<float2 *>(out + (size_t)(q + j) * kM + 2 * tid), acc[j]);
                    ssum = fmaf(acc[j].x, acc[j].x, ssum);
                    ssum = fmaf(acc[j].y, acc[j].y, ssum);
                    smax = fmaxf(smax, fmaxf(fabsf(acc[j].x), fabsf(acc[j].y)));
                }
            }
        }
        dsum += (double)ssum;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) smax = fmaxf(smax, __shfl_xor_sync(0xffffffffu, smax, o));
        if (lane == 0) sred[warp] = smax;

        if (is_last && q + kStep >= qe) {
            // carry the last 15 valid slices: relative slice i = nvalid-15 .. nvalid-1 of this step
            float *h = a.hist_out + (size_t)series * (kP - 1) * kM;
            for (int idx = 0; idx < kP - 1; ++idx) {
                const int i = nvalid - (kP - 1) + idx;
                const float2 v = (i < 0) ? prev[(kStep + i) * kRow + pn] : cur[i * kRow + pn];
                *reinterpret_cast<float2 *>(h + (size_t)idx * kM + 2 * tid) = v;
            }
        }
        __syncthreads();
        if (tid == 0) {
            float m = sred[0];
#pragma unroll
            for (int w = 1; w < kThreads / 32; ++w) m = fmaxf(m, sred[w]);
            a.chunkmax[(size_t)series * a.chunkmax_pitch + a.step0 + q / kStep] = m;
        }
        float2 *t = prev; prev = cur; cur = t;
    }

    // per-CTA sum of squares, fixed reduction order
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) dsum += __shfl_xor_sync(0xffffffffu, dsum, o);
    if (lane == 0) sdred[warp] = dsum;
    __syncthreads();
    if (tid == 0) {
        double s = 0.0;
        for (int w = 0; w < kThreads / 32; ++w) s += sdred[w];
        a.partial[(size_t)series * a.partial_pitch + a.partial0 + span] = s;
    }
}

}  // namespace

int ippf_configure()
{
    cudaError_t e = cudaFuncSetAttribute(ippf_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes);
    return e == cudaSuccess ? 0 : -1;
}

int launch_ippf(const IppfArgs &a, cudaStream_t st)
{
    if (a.nc <= 0) return 0;
    dim3 grid((unsigned)(a.nseries * a.nspans));
    ippf_kernel<<<grid, kThreads, kSmemBytes, st>>>(a);
    return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

}  // namespace lofar
