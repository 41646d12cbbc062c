// beamform.cu -- step a1/a2: tied-array beamforming fused with the de-dispersion phase.
//
//   Z[b][k][q] = sum_s W[b,s,k] * (X[s,0,k,q] + X[s,1,k,q])            (section 3:
//   "the signal of each station has to be summed with a complex weight given by the station
//   position and the beam direction"; the de-dispersion weight of PAPER.md:52 is folded into W
//   when there is one STEC trial, BASELINE.json:north_star w[b,s,sb]).
//
// The weight has no polarisation index (reading A5), so the two polarisations are added as
// integers first: 8*S*B + 2*S flop per (k,q) instead of 16*S*B.
//
// SIMT fp32 version: one thread owns NT consecutive slices of one sub-band and BT beams in
// registers; a warp reads 32*NT consecutive complex samples of each (station, pol) row, i.e.
// whole 128-byte lines; the S*BT weights of the block's sub-band sit in shared memory and are
// read as warp-wide broadcasts.
#include "plan.h"

namespace lofar {
namespace {

constexpr int kBfThreads = 128;

__device__ __forceinline__ float int_to_float_exact(int v)
{
    // exact for |v| < 2^22: 1.5*2^23 + v is representable, subtracting the bias is exact
    return __int_as_float(0x4B400000 + v) - 12582912.0f;
}

// Load NT complex samples of one (station, pol) row and return them as ints (re, im interleaved).
template <int NT, bool I16>
__device__ __forceinline__ void load_row(const void *row, long long t, int nvalid, int *out)
{
    if (nvalid >= NT) {
        if constexpr (I16) {
            const short *p = reinterpret_cast<const short *>(row) + 2 * t;
            if constexpr (NT == 8) {
                int4 a = __ldg(reinterpret_cast<const int4 *>(p));
                int4 b = __ldg(reinterpret_cast<const int4 *>(p) + 1);
                int w[8] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w};
#pragma unroll
                for (int i = 0; i < 8; ++i) { out[2 * i] = (short)(w[i] & 0xffff); out[2 * i + 1] = w[i] >> 16; }
            } else if constexpr (NT == 4) {
                int4 a = __ldg(reinterpret_cast<const int4 *>(p));
                int w[4] = {a.x, a.y, a.z, a.w};
#pragma unroll
                for (int i = 0; i < 4; ++i) { out[2 * i] = (short)(w[i] & 0xffff); out[2 * i + 1] = w[i] >> 16; }
            } else {
                int2 a = __ldg(reinterpret_cast<const int2 *>(p));
                int w[2] = {a.x, a.y};
#pragma unroll
                for (int i = 0; i < 2; ++i) { out[2 * i] = (short)(w[i] & 0xffff); out[2 * i + 1] = w[i] >> 16; }
            }
        } else {
            const signed char *p = reinterpret_cast<const signed char *>(row) + 2 * t;
            if constexpr (NT == 8) {
                int4 a = __ldg(reinterpret_cast<const int4 *>(p));
                int w[4] = {a.x, a.y, a.z, a.w};
#pragma unroll
                for (int i = 0; i < 16; ++i) out[i] = (signed char)((w[i >> 2] >> (8 * (i & 3))) & 0xff);
            } else if constexpr (NT == 4) {
                int2 a = __ldg(reinterpret_cast<const int2 *>(p));
                int w[2] = {a.x, a.y};
#pragma unroll
                for (int i = 0; i < 8; ++i) out[i] = (signed char)((w[i >> 2] >> (8 * (i & 3))) & 0xff);
            } else {
                int a = __ldg(reinterpret_cast<const int *>(p));
#pragma unroll
                for (int i = 0; i < 4; ++i) out[i] = (signed char)((a >> (8 * i)) & 0xff);
            }
        }
    } else {
#pragma unroll
        for (int i = 0; i < NT; ++i) {
            int re = 0, im = 0;
            if (i < nvalid) {
                if constexpr (I16) {
                    const short *p = reinterpret_cast<const short *>(row) + 2 * (t + i);
                    re = p[0]; im = p[1];
                } else {
                    const signed char *p = reinterpret_cast<const signed char *>(row) + 2 * (t + i);
                    re = p[0]; im = p[1];
                }
            }
            out[2 * i] = re; out[2 * i + 1] = im;
        }
    }
}

template <int BT, int NT, bool I16>
__global__ void __launch_bounds__(kBfThreads) beamform_kernel(BeamformArgs a)
{
    extern __shared__ float2 sW[];   // [S][BT]
    const int k = blockIdx.y;
    const int b0 = blockIdx.z * BT;
    for (int i = threadIdx.x; i < a.S * BT; i += kBfThreads) {
        int s = i / BT, bb = i - s * BT;
        float2 w = make_float2(0.f, 0.f);
        if (b0 + bb < a.B) w = a.W[((size_t)k * a.B + (b0 + bb)) * a.S + s];
        sW[i] = w;
    }
    __syncthreads();

    const long long col = ((long long)blockIdx.x * kBfThreads + threadIdx.x) * NT;   // column in Z
    if (col >= a.nt) return;
    const long long t = a.t0 + col;
    const long long left = a.nt - col;
    const int nvalid = left < NT ? (int)left : NT;
    const size_t esize = I16 ? 4 : 2;   // bytes per complex sample

    float2 acc[BT][NT];
#pragma unroll
    for (int bb = 0; bb < BT; ++bb)
#pragma unroll
        for (int i = 0; i < NT; ++i) acc[bb][i] = make_float2(0.f, 0.f);

    const char *Xb = reinterpret_cast<const char *>(a.X);
    const size_t row_bytes = (size_t)a.xpitch * esize;
#pragma unroll 2
    for (int s = 0; s < a.S; ++s) {
        const char *r0 = Xb + ((size_t)(2 * s) * a.K + k) * row_bytes;
        const char *r1 = Xb + ((size_t)(2 * s + 1) * a.K + k) * row_bytes;
        int v0[2 * NT], v1[2 * NT];
        load_row<NT, I16>(r0, t, nvalid, v0);
        load_row<NT, I16>(r1, t, nvalid, v1);
        float x[2 * NT];
#pragma unroll
        for (int i = 0; i < 2 * NT; ++i) x[i] = int_to_float_exact(v0[i] + v1[i]);
#pragma unroll
        for (int bb = 0; bb < BT; ++bb) {
            const float2 w = sW[s * BT + bb];
#pragma unroll
            for (int i = 0; i < NT; ++i) {
                acc[bb][i].x = fmaf(w.x, x[2 * i], acc[bb][i].x);
                acc[bb][i].x = fmaf(-w.y, x[2 * i + 1], acc[bb][i].x);
                acc[bb][i].y = fmaf(w.x, x[2 * i + 1], acc[bb][i].y);
                acc[bb][i].y = fmaf(w.y, x[2 * i], acc[bb][i].y);
            }
        }
    }

    const bool vec = (NT >= 2) && nvalid == NT && ((a.zpitch & 1) == 0) &&
                     ((reinterpret_cast<size_t>(a.Z) & 15) == 0);
    const int nph = a.nphase > 0 ? a.nphase : 1;
#pragma unroll
    for (int bb = 0; bb < BT; ++bb) {
        if (b0 + bb >= a.B) break;
        for (int d = 0; d < nph; ++d) {
            float2 o[NT];
            if (a.nphase > 0) {
                const float2 ph = a.Dph[(size_t)d * a.K + k];
#pragma unroll
                for (int i = 0; i < NT; ++i) o[i] = make_float2(ph.x * acc[bb][i].x - ph.y * acc[bb][i].y,
                                                               ph.x * acc[bb][i].y + ph.y * acc[bb][i].x);
            } else {
#pragma unroll
                for (int i = 0; i < NT; ++i) o[i] = acc[bb][i];
            }
            float2 *zr = a.Z + ((size_t)((b0 + bb) * nph + d) * a.K + k) * (size_t)a.zpitch + col;
            if (vec) {
#pragma unroll
                for (int i = 0; i < NT; i += 2)
                    *reinterpret_cast<float4 *>(zr + i) = make_float4(o[i].x, o[i].y, o[i + 1].x, o[i + 1].y);
            } else {
#pragma unroll
                for (int i = 0; i < NT; ++i)
                    if (i < nvalid) zr[i] = o[i];
            }
        }
    }
}

template <int BT, int NT>
int launch_bt(const BeamformArgs &a, cudaStream_t st)
{
    dim3 grid((unsigned)((a.nt + (long long)kBfThreads * NT - 1) / ((long long)kBfThreads * NT)),
              (unsigned)a.K, (unsigned)((a.B + BT - 1) / BT));
    size_t smem = (size_t)a.S * BT * sizeof(float2);
    if (a.dtype == LOFAR_CI16)
        beamform_kernel<BT, NT, true><<<grid, kBfThreads, smem, st>>>(a);
    else
        beamform_kernel<BT, NT, false><<<grid, kBfThreads, smem, st>>>(a);
    return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

}  // namespace

int launch_beamform(const BeamformArgs &a, cudaStream_t st)
{
    if (a.nt <= 0) return 0;
    if (a.B == 1) return launch_bt<1, 8>(a, st);
    if (a.B == 2) return launch_bt<2, 8>(a, st);
    if (a.B <= 4) return launch_bt<4, 8>(a, st);
    if (a.B <= 8) return launch_bt<8, 4>(a, st);
    if (a.B <= 12) return launch_bt<12, 4>(a, st);
    return launch_bt<24, 2>(a, st);
}

}  // namespace lofar
