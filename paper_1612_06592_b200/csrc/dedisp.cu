// dedisp.cu -- row f2 of SURVEY.md 8(f): exact, paper-order de-dispersion of the reconstructed 5 ns series
// (section 3: "the signal is Fourier transformed, multiplied in frequency domain by a complex weight
// depending on the STEC value and then transformed back"; reading A24 in DESIGN.md).
//
// Overlap-save: one CTA takes a segment of 16 slices (16384 real samples) of one beam, transforms it, multiplies
// bin j by D[j] = exp(-2 pi i 1.343e9 STEC / f_j), f_j = f_zone + j clock / 16384, transforms back and keeps the
// 14 slices in the middle (the de-dispersion chirp of the band is shorter than the one-slice guard).  The output
// runs one slice behind the input.
//
// The 16384-point real transform is an 8192-point complex one on z[n] = x[2n] + i x[2n+1], done as 16 x 512 in
// shared memory with the two building blocks of the inverse polyphase filter (idft16p, fft512_warp):
//   forward (as the conjugate of an inverse transform of conj z):
//     thread n2: 16-point DFT over n1 of z[512 n1 + n2], twiddle exp(2 pi i n2 k1 / 8192) -> rows[k1][n2];
//     warp k1 : 512-point FFT of row k1 -> element k = k1 + 16 k2 at rows[k1][k2];
//   pair stage: thread owns bins (j, 8192-j): real-transform split, multiplication by D, merge for the way back;
//   inverse : warp k1: 512-point FFT of row k1; thread n2: twiddle, 16-point DFT over k1 -> slice n1, pair n2.
// Input slice n1 of a segment is a contiguous row of 512 float2 for the threads n2: coalesced both ways.
#include "fft_warp.cuh"
#include "plan.h"

namespace lofar {
namespace {

constexpr int kDdThreads = 512;
constexpr int kSeg = 16, kKeep = 14;       // slices per segment, slices kept (one guard slice at either end)
constexpr int kNc = 8192;                  // complex transform length
constexpr int kDdRow = 545;                // float2 per row: pad(511) = 542 < 545
constexpr size_t kDdSmem = (size_t)(kSeg * kDdRow + 256 + 512) * sizeof(float2);

__device__ __forceinline__ float2 cmulf(float2 a, float2 b) { return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ float2 conjf(float2 a) { return make_float2(a.x, -a.y); }

// Twiddle exp(2 pi i tid k1 / 8192) of the 16 x 512 split, k1 = 0..15, from its four binary powers b[i] =
// exp(2 pi i tid 2^i / 8192): four table loads per thread (strides 1, 2, 4, 8) and at most three products instead of
// sixteen loads whose stride grows with k1 -- those loads were half of the kernel's L1 traffic (ncu: l1tex 78 % busy).
template <int K1>
__device__ __forceinline__ float2 tw_pow(const float2 (&b)[4])
{
    float2 w = make_float2(1.f, 0.f);
    bool have = false;
#pragma unroll
    for (int i = 0; i < 4; ++i)
        if (K1 & (1 << i)) { w = have ? cmulf(w, b[i]) : b[i]; have = true; }
    return w;
}
template <int K1, typename F>
__device__ __forceinline__ void for_k1(F &&f, const float2 (&b)[4])
{
    f(K1, tw_pow<K1>(b));
    if constexpr (K1 < 15) for_k1<K1 + 1>(f, b);
}

// Position of transform element k = k1 + 16 k2 in the rows.
__device__ __forceinline__ int pos(int k) { return (k & 15) * kDdRow + pad(k >> 4); }

__global__ void __launch_bounds__(kDdThreads, 2) dedisp_kernel(DedispArgs a)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2 *rows = reinterpret_cast<float2 *>(smem_raw);          // [16][kDdRow]
    float2 *stw = rows + kSeg * kDdRow;                            // fft512_warp reads its twiddles at stw + 256
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int seg = blockIdx.x, series = blockIdx.y;
    const int beam = series / a.D, d = series - beam * a.D;
    for (int i = tid; i < 512; i += kDdThreads) stw[256 + i] = a.tw512[i];

    // ---- forward, step 1: thread n2 = tid ----
    const long long s0 = (long long)seg * kKeep;                   // first input slice (xlead coordinates)
    const float *xin = a.xlead + (size_t)beam * a.xpitch;
    u64 x[16];
#pragma unroll
    for (int n1 = 0; n1 < 16; ++n1) {
        float2 v = make_float2(0.f, 0.f);
        if (s0 + n1 < a.nlead) v = *reinterpret_cast<const float2 *>(xin + (size_t)(s0 + n1) * kM + 2 * tid);
        x[n1] = PK(v.x, -v.y);                                      // conj z
    }
    idft16p(x);
    float2 bw[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) bw[i] = __ldg(a.tw8192 + ((tid << i) & (kNc - 1)));
    {
        float2 *col = rows + pad(tid);
        for_k1<0>([&](int k1, float2 w) { sts64(col + k1 * kDdRow, cmulp(x[k1], w.x, w.y)); }, bw);
    }
    __syncthreads();
    fft512_warp(rows + warp * kDdRow, stw, lane);                  // rows now hold conj(FFT z)
    __syncthreads();

    // ---- pair stage: bins (j, N-j), j = 1 .. N/2; bin 0 carries the two real bins 0 and N ----
    const float2 *Dt = a.Dtab + (size_t)d * (kNc + 1);
    for (int j = tid; j <= kNc / 2; j += kDdThreads) {
        if (j == 0) {
            const float2 z0 = conjf(rows[pos(0)]);
            const float y0 = (z0.x + z0.y) * Dt[0].x, yn = (z0.x - z0.y) * Dt[kNc].x;
            rows[pos(0)] = make_float2(y0 + yn, y0 - yn);
            continue;
        }
        const float2 A = conjf(rows[pos(j)]), B = conjf(rows[pos(kNc - j)]);
        const float2 wj = conjf(__ldg(a.tw16k + j));                // exp(-2 pi i j / 16384)
        // X[j] = (A + conj B)/2 - (i/2) w_j (A - conj B);  X[N-j] = (B + conj A)/2 + (i/2) conj(w_j) (B - conj A)
        const float2 sp = make_float2(0.5f * (A.x + B.x), 0.5f * (A.y - B.y));
        const float2 df = make_float2(0.5f * (A.x - B.x), 0.5f * (A.y + B.y));
        const float2 wd = cmulf(wj, df);                            // w_j (A - conj B)/2
        const float2 Xj = make_float2(sp.x + wd.y, sp.y - wd.x);    // sp - i wd
        const float2 Xn = make_float2(sp.x - wd.y, -sp.y - wd.x);   // conj(sp) + i conj(w_j) conj(-df) = conj(sp + i wd)
        const float2 Yj = cmulf(Xj, __ldg(Dt + j)), Yn = cmulf(Xn, __ldg(Dt + kNc - j));
        // V[j] = (Y[j] + conj Y[N-j]) + i conj(w_j) (Y[j] - conj Y[N-j]);  V[N-j] = conj(P) + i (-w_j) conj(-Q) ...
        const float2 P = make_float2(Yj.x + Yn.x, Yj.y - Yn.y);
        const float2 Q = make_float2(Yj.x - Yn.x, Yj.y + Yn.y);
        const float2 wq = cmulf(conjf(wj), Q);
        rows[pos(j)] = make_float2(P.x - wq.y, P.y + wq.x);          // P + i wq
        if (j != kNc / 2) rows[pos(kNc - j)] = make_float2(P.x + wq.y, -P.y + wq.x);   // conj(P - i wq)
    }
    __syncthreads();

    // ---- inverse, step 1: warp k1; step 2: thread n2 ----
    fft512_warp(rows + warp * kDdRow, stw, lane);
    __syncthreads();
#pragma unroll
    for (int i = 0; i < 4; ++i) bw[i] = __ldg(a.tw8192 + ((tid << i) & (kNc - 1)));
    {
        const float2 *col = rows + pad(tid);
        for_k1<0>([&](int k1, float2 w) { const float2 v = col[k1 * kDdRow]; x[k1] = cmulp(PK(v.x, v.y), w.x, w.y); }, bw);
    }
    idft16p(x);
    const float scale = 1.0f / 16384.0f;
    float *out = a.series + (size_t)series * a.series_pitch;
#pragma unroll
    for (int n1 = 1; n1 <= kKeep; ++n1) {
        const long long q = s0 + n1 - 1;                            // output slice: one slice behind the input
        if (q < a.T) *reinterpret_cast<float2 *>(out + (size_t)q * kM + 2 * tid) = make_float2(LO(x[n1]) * scale, HI(x[n1]) * scale);
    }
}

}  // namespace

int dedisp_configure()
{
    cudaError_t e = cudaFuncSetAttribute(dedisp_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kDdSmem);
    return e == cudaSuccess ? 0 : -1;
}

int launch_dedisp(const DedispArgs &a, cudaStream_t st)
{
    if (a.T <= 0) return 0;
    dim3 grid((unsigned)((a.T + kKeep - 1) / kKeep), (unsigned)(a.B * a.D));
    dedisp_kernel<<<grid, kDdThreads, kDdSmem, st>>>(a);
    return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

}  // namespace lofar
