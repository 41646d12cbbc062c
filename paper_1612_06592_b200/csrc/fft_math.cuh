// fft_math.cuh -- small complex helpers and the index maps of the 1024-point C2R inverse FFT
// (step a3, "an inverse Fourier transformation F^-1 y~ = y").
//
// The 1024-point Hermitian inverse transform of one time slice is computed as one 512-point
// complex inverse FFT (a radix-16 pass and a radix-32 pass, one shared-memory exchange between them) of
//     V[k] = (Y[k] + conj(Y[512-k])) + i w^k (Y[k] - conj(Y[512-k])),   w = exp(2 pi i / 1024),
// whose output v[n] = y[2n] + i y[2n+1] is the real series in natural order.
// Everything here is __host__ __device__ so that the index logic can be exercised on the CPU
// build box; none of it is shared with oracle/.
#pragma once
#include <cuda_runtime.h>

#ifndef LOFAR_HD
#define LOFAR_HD __host__ __device__ __forceinline__
#endif

namespace lofar {

constexpr int kM = 1024;      // PPF / FFT size (real points per slice)
constexpr int kH = 512;       // complex FFT length, half spectrum bins 0..511
constexpr int kP = 16;        // taps per polyphase branch
constexpr int kStep = 16;     // slices per processing step (one 128-byte line of float2 per sub-band row)
constexpr int kRow = 545;     // float2 per slice row in shared memory: pad(511) = 542 < 545, 545 = 1 (mod 8)

// (Packed FADD2/FFMA2 were measured and dropped: FFMA2 sustains 70 FMA/clk/SM against 113 for scalar FFMA.)
LOFAR_HD float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
LOFAR_HD float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
LOFAR_HD float2 cmul(float2 a, float2 b) { return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
LOFAR_HD float2 cconj(float2 a) { return make_float2(a.x, -a.y); }
LOFAR_HD float2 cmuli(float2 a) { return make_float2(-a.y, a.x); }   // i * a

// Shared-memory index of complex element i of a slice row: one pad slot per 16 elements keeps the
// stride-64 reads conflict-free and the strided Stockham writes at most 2-way conflicted.
LOFAR_HD int pad(int i) { return i + (i >> 4); }

// Pre-pass for one conjugate pair (m, 512-m), 1 <= m <= 255.
//   a = Y[m], b = Y[512-m], w = exp(2 pi i m / 1024).
//   P = a + conj(b), U = i w (a - conj(b));  V[m] = P + U,  V[512-m] = conj(P - U).
LOFAR_HD void prepass_pair(float2 a, float2 b, float2 w, float2 &vm, float2 &vmirror)
{
    float2 p = cadd(a, cconj(b));
    float2 u = cmuli(cmul(w, csub(a, cconj(b))));
    vm = cadd(p, u);
    vmirror = cconj(csub(p, u));
}
// The two self-paired bins: V[0] = Re(Y[0]) (1 + i) (bin 512 is always zero, reading A10) and
// V[256] = 2 conj(Y[256]).
LOFAR_HD float2 prepass_dc(float2 y0) { return make_float2(y0.x, y0.x); }
LOFAR_HD float2 prepass_quarter(float2 y256) { return make_float2(2.0f * y256.x, -2.0f * y256.y); }

// Inverse 8-point DFT in place: x[m] <- sum_r x[r] exp(+2 pi i r m / 8).
LOFAR_HD void idft8(float2 *x)
{
    const float s = 0.70710678118654752440f;
    // even part: 4-point inverse DFT of x0,x2,x4,x6; odd part of x1,x3,x5,x7
    float2 a0 = cadd(x[0], x[4]), a1 = csub(x[0], x[4]);
    float2 a2 = cadd(x[2], x[6]), a3 = cmuli(csub(x[2], x[6]));
    float2 e0 = cadd(a0, a2), e2 = csub(a0, a2), e1 = cadd(a1, a3), e3 = csub(a1, a3);
    float2 b0 = cadd(x[1], x[5]), b1 = csub(x[1], x[5]);
    float2 b2 = cadd(x[3], x[7]), b3 = cmuli(csub(x[3], x[7]));
    float2 o0 = cadd(b0, b2), o2 = csub(b0, b2), o1 = cadd(b1, b3), o3 = csub(b1, b3);
    // twiddles W8^m = exp(+i pi m / 4) on the odd part
    float2 t1 = make_float2(s * (o1.x - o1.y), s * (o1.x + o1.y));   // o1 * (1+i)/sqrt2
    float2 t2 = cmuli(o2);                                            // o2 * i
    float2 t3 = make_float2(-s * (o3.x + o3.y), s * (o3.x - o3.y));  // o3 * (-1+i)/sqrt2
    x[0] = cadd(e0, o0); x[4] = csub(e0, o0);
    x[1] = cadd(e1, t1); x[5] = csub(e1, t1);
    x[2] = cadd(e2, t2); x[6] = csub(e2, t2);
    x[3] = cadd(e3, t3); x[7] = csub(e3, t3);
}

// Inverse 16-point DFT in place (two 8-point DFTs of the even / odd inputs, then the W16^m butterflies).
LOFAR_HD void idft16(float2 *x)
{
    float2 e[8], o[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) { e[i] = x[2 * i]; o[i] = x[2 * i + 1]; }
    idft8(e);
    idft8(o);
    const float c1 = 0.92387953251128675613f, s1 = 0.38268343236508977173f, h = 0.70710678118654752440f;
    const float wc[8] = {1.f, c1, h, s1, 0.f, -s1, -h, -c1};
    const float ws[8] = {0.f, s1, h, c1, 1.f, c1, h, s1};
#pragma unroll
    for (int m = 0; m < 8; ++m) {
        const float2 t = m == 0 ? o[0] : (m == 4 ? cmuli(o[4]) : cmul(o[m], make_float2(wc[m], ws[m])));
        x[m] = cadd(e[m], t);
        x[m + 8] = csub(e[m], t);
    }
}

// Stockham pass with sub-transform length Ns (1, 8, 64): butterfly j (0..63) reads elements
// j + 64 r, r = 0..7, multiplies element r by exp(+2 pi i (j mod Ns) r / (8 Ns)) and writes output m
// to (j / Ns) * 8 Ns + (j mod Ns) + m Ns.
LOFAR_HD int stockham_src(int j, int r) { return j + 64 * r; }
LOFAR_HD int stockham_dst(int j, int m, int Ns) { return (j / Ns) * (8 * Ns) + (j % Ns) + m * Ns; }

}  // namespace lofar
