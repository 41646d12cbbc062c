// fft_math.cuh -- constants, the shared-memory index map and the self-paired bins of the 1024-point C2R inverse FFT
// (step a3, "an inverse Fourier transformation F^-1 y~ = y").
//
// The 1024-point Hermitian inverse transform of one time slice is computed as one 512-point
// complex inverse FFT (a radix-16 pass and a radix-32 pass, one shared-memory exchange between them) of
//     V[k] = (Y[k] + conj(Y[512-k])) + i w^k (Y[k] - conj(Y[512-k])),   w = exp(2 pi i / 1024),
// whose output v[n] = y[2n] + i y[2n+1] is the real series in natural order.
// The pair pre-pass and the radix-16 / radix-32 passes are in ippf.cu (packed fp32x2 arithmetic).
// None of this is shared with oracle/.
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

// Shared-memory index of complex element i of a slice row: one pad slot per 16 elements keeps the
// stride-16 writes of the radix-16 pass conflict-free.
LOFAR_HD int pad(int i) { return i + (i >> 4); }

// The two self-paired bins of the pre-pass: V[0] = Re(Y[0]) (1 + i) (bin 512 is always zero, reading A10)
// and V[256] = 2 conj(Y[256]).
LOFAR_HD float2 prepass_dc(float2 y0) { return make_float2(y0.x, y0.x); }
LOFAR_HD float2 prepass_quarter(float2 y256) { return make_float2(2.0f * y256.x, -2.0f * y256.y); }

}  // namespace lofar
