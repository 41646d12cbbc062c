// ippf.cu -- steps a3 + a4 (+ the sum of squares and per-step maximum that a5 needs):
// inversion of the polyphase filter bank (section 3: "an inverse Fourier
// transformation F^-1 y~ = y of the filtered signal" followed by the FIR system H; here one
// application of the matched synthesis FIR g = 1024 h, reading A8).
//
// One CTA (512 threads, 16 warps, one per SM) owns one series and marches along a span of time slices in
// steps of 16 slices:
//   stage    : the K selected sub-band rows of the step -- one 128-byte line per row -- are brought into a
//              shared-memory stage by bulk asynchronous copies (cp.async.bulk + mbarrier; one copy of
//              K*128 bytes from the plan's tiled scratch, one copy per row from a caller's Z), issued one
//              step ahead so that they fly during the FFT and FIR of the current step;
//   pass A   : thread (bin residue j mod 32, slice t) reads its 16 bins j + 32 r and their mirrors from the stage,
//              applies the trial phasor if asked, forms the packed half-spectrum V of the real transform
//              (fft_math.cuh), does the radix-16 butterflies over r, applies the radix-32 twiddles and stores the
//              result slice-major into the current slice buffer (V itself is never written);
//   pass B   : warp w finishes slice w in place: the radix-32 pass of 512 = 16 x 32 (fft512_pass_b);
//   FIR      : thread n owns output residues r = 2n, 2n+1 and keeps their 16 tap pairs in registers; the
//              31-slice window (15 carried + 16 new) is read from the previous and current slice buffers;
//              16 x 1024 contiguous output samples are written per step.
// The transform's complex adds and butterflies are packed fp32x2 instructions (FADD2 / FFMA2: half the issue slots in
// phases that are issue-bound); the FIR is scalar FFMA (the packed form with three distinct register operands is
// register-file limited). Launch parameters are read from the constant bank where they are used and slice indices
// are 32-bit, which keeps the persistent register state small: the kernel sits at the 128-register cap and every
// register the scheduler gets back shows in the FIR.
// Synchronisation per step: one full barrier (after pass A: every warp writes into every slice row) and two split
// ones on mbarriers -- warps arrive after pass B and the FIR waits only before it reads the first row of the current
// step (the 15 carried rows are applied first); warps arrive after the FIR and pass A waits only before its stores.
// The 15-slice history lives in the "previous" buffer, is loaded from the plan at the start of a block and
// written back by the CTA that owns the last span; CTAs that start in the middle of a block first
// transform the 16 slices before their span (no output).
#include "fft_warp.cuh"
#include "plan.h"

namespace lofar {
namespace {

constexpr int kThreads = 512;
constexpr int kTwCount = 256 + 512;        // w1024[256], TB[32][16] = exp(2 pi i j r / 512)
constexpr int kStageF2 = (kH + 1) * kStep; // stage: bins 0..512 x 16 slices of float2 (row 512 stays zero)
constexpr size_t kSmemBytes = (size_t)(2 * kStep * kRow + kStageF2 + kTwCount + kH + 1) * sizeof(float2) + 256;

// ---- mbarrier + bulk asynchronous copy (TMA unit, SASS UBLKCP / SYNCS) ------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" :: "r"(bar) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    while (!mbar_try_wait(bar, parity)) {}
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 :: "r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}

// Brings the K rows x 16 slices of the step starting at slice q into rows k0 .. k0 + K - 1 of the stage (`stage` points at row k0).
// Zs: this series' beam sums. Returns true if the copy is asynchronous (completion on the mbarrier), false if the
// threads stored it. The launch parameters are read where they are used (constant bank), not kept in registers.
__device__ __forceinline__ bool stage_fill(const IppfArgs &a, const float2 *Zs, int q, float2 *stage, uint32_t bar, int tid)
{
    if (a.ztile) {
        // plan scratch [tile = q/16][K][16]: the whole step is one contiguous block
        if (tid == 0) {
            const uint32_t bytes = (uint32_t)a.K * 128u;
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // the stage was last read by ordinary loads
            mbar_arrive_expect_tx(bar, bytes);
            bulk_g2s(smem_u32(stage), Zs + (size_t)(q >> 4) * a.K * 16, bytes, bar);
        }
        return true;
    }
    if (a.vec_ok && q + kStep <= a.nc) {
        // caller's Z [K][zpitch]: one 128-byte line per row
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        if (tid == 0) mbar_arrive_expect_tx(bar, (uint32_t)a.K * 128u);
        for (int j = tid; j < a.K; j += kThreads)
            bulk_g2s(smem_u32(stage + j * kStep), Zs + (size_t)j * a.zpitch + q, 128u, bar);
        return true;
    }
    // ragged or unaligned: plain loads, zero beyond the end of the launch
    for (int idx = tid; idx < a.K * kStep; idx += kThreads) {
        const int j = idx >> 4, t = idx & 15;
        float2 v = make_float2(0.f, 0.f);
        if (q + t < a.nc) v = Zs[(size_t)j * a.zpitch + q + t];
        stage[idx] = v;
    }
    return false;
}

// Twiddles into shared memory: w1024[j + 32 r] goes to stw[8 j + r] (the 8 values a pass-A thread needs side by side),
// the radix-32 table TBs[32][16] follows unchanged at stw + 256.
__device__ __forceinline__ void load_twiddles(float2 *stw, const float2 *tw, int tid)
{
    for (int i = tid; i < kTwCount; i += kThreads) stw[i < 256 ? 8 * (i & 31) + (i >> 5) : i] = tw[i];
}

// ---- pass A: pair pre-pass fused with the radix-16 pass of the 512-point transform ---------------------
// The stage is indexed by the absolute bin: row m holds the 16 slices of bin m; the rows of unselected bins are
// zeroed once per CTA (reading A10) and the copies only ever write rows k0 .. k0 + K - 1, so the transform reads
// it without bounds tests. The STEC trial phasor (a2, sph[m]) multiplies a beam sum as it enters the transform.
template <bool PH>
__device__ __forceinline__ u64 ldz(const float2 *p, const float2 *ph)
{
    const u64 v = lds64(p);
    if (!PH) return v;
    const float2 f = *ph;
    return cmulp(v, f.x, f.y);
}

// One conjugate pair: a = Y[m], b = Y[512-m], w = exp(2 pi i m / 1024):
//   P = a + conj(b), D = a - conj(b), U' = (Im(wD), Re(wD));  V[m] = (P.x - U'.x, P.y + U'.y),
//   V[512-m] = (P.x + U'.x, U'.y - P.y)                                 (fft_math.cuh)
__device__ __forceinline__ void vpair(u64 a, u64 b, float2 w, u64 &vm, u64 &vmir)
{
    const u64 pm = PK(1.f, -1.f), mp = PK(-1.f, 1.f);
    const u64 P = fma2(b, pm, a), D = fma2(b, mp, a);
    const float dx = LO(D), dy = HI(D);
    const u64 U = PK(fmaf(w.x, dy, w.y * dx), fmaf(w.x, dx, -w.y * dy));
    vm = fma2(U, mp, P);
    vmir = fma2(P, pm, U);
}

// All 512 threads, one step: thread (j, t) -- j = residue of the bin index mod 32, t = slice of the step -- builds
// V[j + 32 r], r = 0..15, of its slice straight from the stage ([513][16], so the 16 slices of a half-warp read one
// 128-byte line), does the 16-point DFT over r, applies the radix-32 twiddles exp(2 pi i j m / 512) and stores
// the result slice-major at dst[t][pad(16 j + m)]. The mirror of bin j + 32 r is bin (32 - j) + 32 (15 - r): a
// warp holds j in its low and 32 - j in its high half, each thread forms the pairs r = 0..7 and hands the
// mirrored values to its partner lane (shuffle). Warp 0 holds the two self-paired residues j = 0 and j = 16: the same
// code with the lane itself as partner; for j = 0 the pairs are (32 r, 32 (16 - r)), i.e. the mirrored values land one
// place further (fixed up below), bin 0 keeps its real part only and pairs with the always-zero row 512 (reading A10),
// and bin 256 is its own mirror. One code path for all warps keeps the loop body inside the instruction cache.
template <bool PH>
__device__ __forceinline__ void pass_a(const float2 *stage, const float2 *sph, float2 *dst, const float2 *stw, int tid,
                                       uint32_t bar_f = 0, uint32_t phase_f = 0)
{
    const int warp = tid >> 5, lane = tid & 31, half = lane >> 4, t = lane & 15;
    constexpr int R = 32 * kStep;                  // stage elements between bins m and m + 32
    const int j = half ? (warp ? 32 - warp : 16) : warp;
    const bool dc = (warp | half) == 0;            // the thread that holds bins 0, 32, ..., 480
    u64 x[16];
    const float2 *sa = stage + j * kStep + t, *sb = stage + (512 - j) * kStep + t;
    const float2 *pa = sph + j, *pb = sph + 512 - j;
    // the 8 pair twiddles w^(j + 32 r) of this thread sit side by side (load_twiddles) and come in as four 16-byte loads
    float2 wj[8];
    {
        const float4 *w4 = reinterpret_cast<const float4 *>(stw + 8 * j);
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const float4 v = w4[r];
            wj[2 * r] = make_float2(v.x, v.y);
            wj[2 * r + 1] = make_float2(v.z, v.w);
        }
    }
    u64 give[8];
    {
        u64 a0 = ldz<PH>(sa, pa);
        if (dc) a0 = PK(LO(a0), 0.f);
        vpair(a0, ldz<PH>(sb, pb), wj[0], x[0], give[0]);
    }
#pragma unroll
    for (int r = 1; r < 8; ++r) vpair(ldz<PH>(sa + r * R, pa + 32 * r), ldz<PH>(sb - r * R, pb - 32 * r), wj[r], x[r], give[r]);
    const int partner = warp ? lane ^ 16 : lane;
#pragma unroll
    for (int r = 0; r < 8; ++r) x[15 - r] = __shfl_sync(0xffffffffu, give[r], partner);
    if (warp == 0) {
        const u64 y256 = ldz<PH>(stage + 256 * kStep + t, sph + 256);
        if (dc) {
#pragma unroll
            for (int m = 15; m > 8; --m) x[m] = x[m - 1];           // mirror of bin 32 r is bin 32 (16 - r)
            x[8] = PK(2.0f * LO(y256), -2.0f * HI(y256));           // prepass_quarter
        }
    }
    idft16p(x);
    const float2 *T = stw + 256 + 16 * j;          // T[m] = TBs[j][m] = +-exp(2 pi i j m / 512), minus for j = 3 (mod 4)
    float2 *row = dst + t * kRow + 17 * j;         // pad(16 j + m) = 17 j + m
    if ((j & 3) == 3) x[0] = PK(-LO(x[0]), -HI(x[0]));      // TBs[j][0] = -1: the one twiddle that is not loaded
    {
        const float4 *T4 = reinterpret_cast<const float4 *>(T);      // (T[m], T[m + 1]) per 16-byte load; T is 128-byte aligned
#pragma unroll
        for (int m = 0; m < 16; m += 2) {
            const float4 f = T4[m >> 1];
            if (m) x[m] = cmulp(x[m], f.x, f.y);
            x[m + 1] = cmulp(x[m + 1], f.z, f.w);
        }
    }
    // dst still holds the carried rows the FIR of the previous step reads: wait for all warps to be through with it
    // only now, with everything of this step but its 16 stores done (split barrier)
    if (bar_f) mbar_wait(bar_f, phase_f);
#pragma unroll
    for (int m = 0; m < 16; ++m) sts64(row + m, x[m]);
}

// Rare path, kept out of line and out of the FIR's registers: a thread whose step maximum exceeds the threshold
// recomputes its 2 x 16 outputs (taps re-read from global memory) and records every sample above the threshold
// (all trials; the best trial per sample is selected after the sort).
__device__ __noinline__ void emit_step(const float2 *prev, const float2 *cur, const float2 *gs, int tid, int pn, int nvalid,
                                       lofar_candidate *cand, uint32_t *count, uint32_t cap, uint32_t series, uint32_t trial,
                                       float thr, float sigma, uint64_t sample0)
{
    for (int j = 0; j < nvalid; ++j) {
        float2 acc = make_float2(0.f, 0.f);
        for (int t = 0; t < kP; ++t) {
            const int i = (kP - 1) + j - t;                    // window element: prev rows 1..15, cur rows 0..15
            const float2 x = (i < kP - 1) ? prev[(i + 1) * kRow + pn] : cur[(i - (kP - 1)) * kRow + pn];
            const float2 g = __ldg(gs + t * kH + tid);
            acc.x = fmaf(g.x, x.x, acc.x);
            acc.y = fmaf(g.y, x.y, acc.y);
        }
#pragma unroll
        for (int c = 0; c < 2; ++c) {
            const float v = fabsf(c ? acc.y : acc.x);
            if (v > thr) {
                const uint32_t slot = atomicAdd(count, 1u);
                if (slot < cap) {
                    lofar_candidate r;
                    r.series = series; r.trial = trial; r.sample = sample0 + (uint64_t)j * kM + 2 * tid + c;
                    r.env = v; r.sigma = sigma;
                    cand[slot] = r;
                }
            }
        }
    }
}

// One tap of the FIR on a residue pair: two scalar FFMA. The packed FFMA2 (-DLOFAR_FIR_PACKED) takes half the issue
// slots but, with three distinct register operands, is register-file limited to ~79 FMA/clk/SM against ~100 for the
// scalar form (micro-benchmark); measured in the kernel: 6.05 ms scalar, 6.29 ms packed.
__device__ __forceinline__ u64 fir_fma(u64 g, u64 x, u64 acc)
{
#ifdef LOFAR_FIR_PACKED
    return fma2p(g, x, acc);
#else
    return PK(fmaf(LO(g), LO(x), LO(acc)), fmaf(HI(g), HI(x), HI(acc)));
#endif
}

// Synthesis FIR of one step: out[j] = sum_t g[t] * win[15 + j - t], j = 0..15, window = prev rows 1..15 + cur rows
// 0..15, column pn; FULL = all 16 output slices valid (no predicates on the fast path).
template <bool FULL>
__device__ __forceinline__ void fir_step(const float2 *prev, const float2 *cur, const u64 (&g)[kP], int pn, float *out,
                                         int tid, int nvalid, u64 &ssum2, float &smax, uint32_t bar_b = 0, uint32_t phase_b = 0)
{
    u64 acc[kStep];
#pragma unroll
    for (int j = 0; j < kStep; ++j) acc[j] = 0ull;
#pragma unroll
    for (int i = 0; i < kP - 1 + kStep; ++i) {
        // the 15 carried rows need nothing of this step: the warps only wait for each other's radix-32 pass here, with
        // almost half of the FIR's arithmetic already issued (split barrier: arrive after pass B, wait before row 0)
        if (i == kP - 1 && bar_b) mbar_wait(bar_b, phase_b);
        const u64 x = lds64((i < kP - 1) ? prev + (i + 1) * kRow + pn : cur + (i - (kP - 1)) * kRow + pn);
#pragma unroll
        for (int t = 0; t < kP; ++t) {
            const int j = i - (kP - 1) + t;
            if (j >= 0 && j < kStep) acc[j] = fir_fma(g[t], x, acc[j]);
        }
        // output slice j = i - 15 is complete once window element i has been applied: store it now so
        // that the 64 KB of stores per step are spread over the second half of the FIR
        if (i >= kP - 1) {
            const int j = i - (kP - 1);
            if (FULL || j < nvalid) {
                const float vx = LO(acc[j]), vy = HI(acc[j]);
#ifndef LOFAR_ABLATE_STORES
#ifdef LOFAR_ST_PLAIN
                if (out) *reinterpret_cast<float2 *>(out + (size_t)j * kM + 2 * tid) = make_float2(vx, vy);
#else
                if (out) __stcs(reinterpret_cast<float2 *>(out + (size_t)j * kM + 2 * tid), make_float2(vx, vy));   // written once, not re-read here
#endif
#endif
                ssum2 = fma2p(acc[j], acc[j], ssum2);
                smax = fmaxf(smax, fmaxf(fabsf(vx), fabsf(vy)));
            }
        }
    }
}

__global__ void __launch_bounds__(kThreads, 1) ippf_kernel(IppfArgs a)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float2 *stage = reinterpret_cast<float2 *>(smem_raw);          // [512][16] by bin, 128-byte aligned for the bulk copies
    float2 *buf0 = stage + kStageF2;
    float2 *buf1 = buf0 + kStep * kRow;
    float2 *stw = buf1 + kStep * kRow;                             // [kTwCount]
    float2 *sph = stw + kTwCount;                                  // [K] phasors of this series' STEC trial (a2)
    float *sred = reinterpret_cast<float *>(sph + kH + 1);         // 16 floats, 16 doubles, the mbarrier
    double *sdred = reinterpret_cast<double *>(sred + 16);
    const uint32_t bar = smem_u32(sdred + 16);
    const uint32_t bar_b = bar + 8;                                // "radix-32 pass done": one arrival per warp and step
    const uint32_t bar_f = bar + 16;                               // "through with the previous step's rows": the same

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int series = blockIdx.x % a.nseries;
    const int span = blockIdx.x / a.nseries;
    const int nc = (int)a.nc;                    // slices of the launch (an int at the boundary)
    const int qs = span * a.span_len;
    if (qs >= nc) return;
    const int qe = (qs + a.span_len < nc) ? qs + a.span_len : nc;
    const bool is_last = (qe == nc);
    const bool trials = a.zmap_trials != 0;      // the STEC trial phasor multiplies the beam sums on their way in (a2)

    const float2 *Zs = a.Z + (size_t)(trials ? series / a.zmap_trials : series) * a.K * (size_t)a.zpitch;

    if (tid == 0) {
        mbar_init(bar, 1);
        mbar_init(bar_b, kThreads / 32);
        mbar_init(bar_f, kThreads / 32);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    load_twiddles(stw, a.tw, tid);
    for (int i = tid; i < kStageF2; i += kThreads) stage[i] = make_float2(0.f, 0.f);   // unselected bins stay zero
    if (trials) {
        const float2 *ph = a.Dph + (size_t)(series % a.zmap_trials) * a.K;
        sph[tid] = make_float2(1.f, 0.f);
        if (tid == 0) sph[kH] = make_float2(1.f, 0.f);           // the always-zero bin 512
        __syncthreads();
        for (int i = tid; i < a.K; i += kThreads) sph[a.k0 + i] = ph[i];
    }
    float2 *stage_k = stage + a.k0 * kStep;      // the copies write rows k0 .. k0 + K - 1
    u64 g[kP];                                   // the 16 tap pairs of residues 2 tid, 2 tid + 1, for the whole span
#pragma unroll
    for (int t = 0; t < kP; ++t) { const float2 v = __ldg(a.gs + t * kH + tid); g[t] = PK(v.x, v.y); }
    const int pn = pad(tid);

    float2 *prev = buf0, *cur = buf1;
    if (span == 0) {
        const float *h = a.hist_in + (size_t)series * (kP - 1) * kM;
#pragma unroll
        for (int i = 0; i < kP - 1; ++i)
            prev[(i + 1) * kRow + pn] = *reinterpret_cast<const float2 *>(h + (size_t)i * kM + 2 * tid);
    }
    __syncthreads();                             // mbarrier, twiddles and history visible

    // the first step of a span that starts inside the block is a warm-up: transform the 16 slices before it
    const int q_first = span == 0 ? qs : qs - kStep;
    uint32_t phase = 0, phase_b = 0, phase_f = 1;     // phase_f = 1: nothing to wait for before the first step
    int pend = -1;                                   // step whose maximum is still in sred (written out after the next pass A)
    bool async = stage_fill(a, Zs, q_first, stage_k, bar, tid);

    double dsum = 0.0;
    const float thr = a.thr ? a.thr[series] : __int_as_float(0x7f800000);    // +inf: no emission from the epilogue

    for (int q = q_first; q < qe; q += kStep) {
        if (async) { while (!mbar_try_wait(bar, phase)) {} phase ^= 1; }
        else __syncthreads();
#ifndef LOFAR_ABLATE_FFT
        if (trials) pass_a<true>(stage, sph, cur, stw, tid, bar_f, phase_f);
        else pass_a<false>(stage, sph, cur, stw, tid, bar_f, phase_f);
#else
        mbar_wait(bar_f, phase_f);
#endif
        phase_f ^= 1;
        // Thread 0 has waited on bar_f inside pass A: every warp has arrived there, i.e. written its maximum of the
        // previous step into sred; and no warp can write the next one before the barrier below, which needs thread 0.
        if (pend >= 0 && tid == 0) {
            float m = sred[0];
#pragma unroll
            for (int w = 1; w < kThreads / 32; ++w) m = fmaxf(m, sred[w]);
            a.chunkmax[(size_t)series * a.chunkmax_pitch + a.step0 + pend] = m;
        }
        __syncthreads();                         // radix-16 results of all 16 slices in cur, stage free
        pend = -1;
        if (q + kStep < qe) async = stage_fill(a, Zs, q + kStep, stage_k, bar, tid);   // flies during pass B + FIR
#ifndef LOFAR_ABLATE_FFT
        fft512_pass_b<false>(cur + warp * kRow, stw, lane);
#endif
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_b);       // waited for where the rows of this step are first read

        if (q >= qs && a.yout) {
            mbar_wait(bar_b, phase_b);
            // LSMR inversion (f1): hand the inverse-DFT rows to the solver instead of applying the matched FIR
            float *yout = a.yout + (size_t)series * a.yout_pitch + a.out0;
            const int nvalid = (qe - q < kStep) ? qe - q : kStep;
            for (int j = 0; j < nvalid; ++j)
                *reinterpret_cast<float2 *>(yout + (size_t)(q + j) * kM + 2 * tid) = cur[j * kRow + pn];
            if (is_last && q + kStep >= qe) {
                float *h = a.hist_out + (size_t)series * (kP - 1) * kM;
                for (int idx = 0; idx < kP - 1; ++idx) {
                    const int i = nvalid - (kP - 1) + idx;
                    const float2 v = (i < 0) ? prev[(kStep + i) * kRow + pn] : cur[i * kRow + pn];
                    *reinterpret_cast<float2 *>(h + (size_t)idx * kM + 2 * tid) = v;
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_f);
        } else if (q >= qs) {
            const int nvalid = (qe - q < kStep) ? qe - q : kStep;
            u64 ssum2 = 0ull;
            float smax = 0.f;
            float *o = a.series ? a.series + (size_t)series * a.series_pitch + a.out0 + (size_t)q * kM : nullptr;
#ifndef LOFAR_ABLATE_FIR
            if (nvalid == kStep) fir_step<true>(prev, cur, g, pn, o, tid, nvalid, ssum2, smax, bar_b, phase_b);
            else fir_step<false>(prev, cur, g, pn, o, tid, nvalid, ssum2, smax, bar_b, phase_b);
#else
            mbar_wait(bar_b, phase_b);
#endif
            if (smax > thr)
                emit_step(prev, cur, a.gs, tid, pn, nvalid, a.cand, a.count, a.cap, (uint32_t)series, (uint32_t)(series % a.D),
                          thr, a.sigma_ref[series], a.offset + (uint64_t)a.out0 + (uint64_t)q * kM);
            dsum += (double)(LO(ssum2) + HI(ssum2));
#pragma unroll
            for (int s = 16; s > 0; s >>= 1) smax = fmaxf(smax, __shfl_xor_sync(0xffffffffu, smax, s));
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
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_f);   // waited for in the next pass A, before it overwrites the carried rows
            pend = q / kStep;
        }
        else {
            mbar_wait(bar_b, phase_b);           // warm-up step: nothing reads the rows, the buffers swap below
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_f);
        }
        phase_b ^= 1;
        float2 *t = prev; prev = cur; cur = t;
    }

    // per-CTA sum of squares, fixed reduction order
#pragma unroll
    for (int s = 16; s > 0; s >>= 1) dsum += __shfl_xor_sync(0xffffffffu, dsum, s);
    if (lane == 0) sdred[warp] = dsum;
    __syncthreads();
    if (tid == 0 && pend >= 0) {
        float m = sred[0];
#pragma unroll
        for (int w = 1; w < kThreads / 32; ++w) m = fmaxf(m, sred[w]);
        a.chunkmax[(size_t)series * a.chunkmax_pitch + a.step0 + pend] = m;
    }
    if (tid == 0) {
        double s = 0.0;
        for (int w = 0; w < kThreads / 32; ++w) s += sdred[w];
        a.partial[(size_t)series * a.partial_pitch + a.partial0 + span] = s;
    }
}


// ---- series-free two-pass trigger: recompute the flagged steps from X ------------------------------
__device__ __forceinline__ float2 read_cx(const void *X, int dtype, size_t idx)
{
    if (dtype == LOFAR_CI16) {
        const short2 v = reinterpret_cast<const short2 *>(X)[idx];
        return make_float2((float)v.x, (float)v.y);
    }
    const char2 v = reinterpret_cast<const char2 *>(X)[idx];
    return make_float2((float)v.x, (float)v.y);
}

// Beam sums of one beam for the 16 slices starting at q, straight into the stage (plain fp32 sums).
__device__ __forceinline__ void stage_from_x(const RescanArgs &r, int beam, long long q, float2 *stage, int tid)
{
    for (int idx = tid; idx < r.K * kStep; idx += kThreads) {
        const int j = idx >> 4, t = idx & 15;
        float2 acc = make_float2(0.f, 0.f);
        if (q + t < r.T) {
            const float2 *w = r.W + ((size_t)j * r.B + beam) * r.S;
            for (int s = 0; s < r.S; ++s) {
                const size_t i0 = ((size_t)(2 * s) * r.K + j) * (size_t)r.xpitch + (size_t)(q + t);
                const float2 x0 = read_cx(r.X, r.dtype, i0), x1 = read_cx(r.X, r.dtype, i0 + (size_t)r.K * r.xpitch);
                const float xr = x0.x + x1.x, xi = x0.y + x1.y;
                const float2 ww = __ldg(w + s);
                acc.x = fmaf(ww.x, xr, fmaf(-ww.y, xi, acc.x));
                acc.y = fmaf(ww.x, xi, fmaf(ww.y, xr, acc.y));
            }
        }
        stage[idx] = acc;
    }
}

__global__ void __launch_bounds__(kThreads, 1) rescan_kernel(RescanArgs r)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float2 *stage = reinterpret_cast<float2 *>(smem_raw);
    float2 *buf0 = stage + kStageF2;
    float2 *buf1 = buf0 + kStep * kRow;
    float2 *stw = buf1 + kStep * kRow;
    float2 *sph = stw + kTwCount;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t total = *r.nitems < r.items_cap ? *r.nitems : r.items_cap;
    if (blockIdx.x >= total) return;
    load_twiddles(stw, r.tw, tid);
    for (int i = tid; i < kStageF2; i += kThreads) stage[i] = make_float2(0.f, 0.f);
    sph[tid] = make_float2(1.f, 0.f);
    if (tid == 0) sph[kH] = make_float2(1.f, 0.f);
    float2 *stage_k = stage + r.k0 * kStep;
    u64 g[kP];
#pragma unroll
    for (int t = 0; t < kP; ++t) { const float2 v = __ldg(r.gs + t * kH + tid); g[t] = PK(v.x, v.y); }
    const int pn = pad(tid);
    __syncthreads();

    for (uint32_t it = blockIdx.x; it < total; it += gridDim.x) {
        const int beam = r.items[it].x;
        const long long q = (long long)r.items[it].y * kStep;
        for (int d = 0; d < r.D; ++d) {
            const int series = beam * r.D + d;
            const float sig = r.sigma[series], thr = r.kappa * sig;
            if (r.chunkmax[(size_t)series * r.chunkmax_pitch + r.items[it].y] < thr * 0.99999f) continue;
            if (r.D > 1)                               // this trial's phasors (read by pass_a after the next barrier)
                for (int i = tid; i < r.K; i += kThreads) sph[r.k0 + i] = r.Dph[(size_t)d * r.K + i];
            if (q == 0) {
                const float *h = r.hist0 + (size_t)series * (kP - 1) * kM;
#pragma unroll
                for (int i = 0; i < kP - 1; ++i)
                    buf0[(i + 1) * kRow + pn] = *reinterpret_cast<const float2 *>(h + (size_t)i * kM + 2 * tid);
            } else {
                stage_from_x(r, beam, q - kStep, stage_k, tid);
                __syncthreads();
                if (r.D > 1) pass_a<true>(stage, sph, buf0, stw, tid);
                else pass_a<false>(stage, sph, buf0, stw, tid);
                __syncthreads();
                fft512_pass_b<false>(buf0 + warp * kRow, stw, lane);
            }
            __syncthreads();
            stage_from_x(r, beam, q, stage_k, tid);
            __syncthreads();
            if (r.D > 1) pass_a<true>(stage, sph, buf1, stw, tid);
            else pass_a<false>(stage, sph, buf1, stw, tid);
            __syncthreads();
            fft512_pass_b<false>(buf1 + warp * kRow, stw, lane);
            __syncthreads();
            const int nvalid = (r.T - q < kStep) ? (int)(r.T - q) : kStep;
            u64 ssum2 = 0ull;
            float smax = 0.f;
            fir_step<false>(buf0, buf1, g, pn, nullptr, tid, nvalid, ssum2, smax);
            if (smax > thr)
                emit_step(buf0, buf1, r.gs, tid, pn, nvalid, r.cand, r.count, r.cap, (uint32_t)series, (uint32_t)d, thr, sig,
                          r.offset + (uint64_t)q * kM);
            __syncthreads();
        }
    }
}

}  // namespace

int ippf_configure()
{
    cudaError_t e = cudaFuncSetAttribute(ippf_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(rescan_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes);
    return e == cudaSuccess ? 0 : -1;
}

int launch_ippf(const IppfArgs &a, cudaStream_t st)
{
    if (a.nc <= 0) return 0;
    dim3 grid((unsigned)(a.nseries * a.nspans));
    ippf_kernel<<<grid, kThreads, kSmemBytes, st>>>(a);
    return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

int launch_rescan(const RescanArgs &a, int grid, cudaStream_t st)
{
    rescan_kernel<<<grid, kThreads, kSmemBytes, st>>>(a);
    return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

}  // namespace lofar
