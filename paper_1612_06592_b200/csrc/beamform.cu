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

// Raw 32-bit words holding NT complex samples of one (station, pol) row.
template <int NT, bool I16>
struct RowWords { static constexpr int value = NT * (I16 ? 4 : 2) / 4; };

template <int NT, bool I16>
__device__ __forceinline__ void load_raw(const void *row, long long t, int nvalid, int *raw)
{
    constexpr int NW = RowWords<NT, I16>::value;
    const char *p = reinterpret_cast<const char *>(row) + (size_t)t * (I16 ? 4 : 2);
    if (nvalid >= NT) {
        if constexpr (NW >= 4) {
#pragma unroll
            for (int i = 0; i < NW / 4; ++i) {
                const int4 v = __ldg(reinterpret_cast<const int4 *>(p) + i);
                raw[4 * i] = v.x; raw[4 * i + 1] = v.y; raw[4 * i + 2] = v.z; raw[4 * i + 3] = v.w;
            }
        } else if constexpr (NW == 2) {
            const int2 v = __ldg(reinterpret_cast<const int2 *>(p));
            raw[0] = v.x; raw[1] = v.y;
        } else {
            raw[0] = __ldg(reinterpret_cast<const int *>(p));
        }
    } else {
        // ragged tail: assemble the words from single samples, zero beyond the end of the row
#pragma unroll
        for (int w = 0; w < NW; ++w) raw[w] = 0;
        if constexpr (I16) {
            const unsigned short *q = reinterpret_cast<const unsigned short *>(p);
#pragma unroll
            for (int i = 0; i < NT; ++i)
                if (i < nvalid) raw[i] = (int)((unsigned)q[2 * i] | ((unsigned)q[2 * i + 1] << 16));
        } else {
            const unsigned char *q = reinterpret_cast<const unsigned char *>(p);
#pragma unroll
            for (int i = 0; i < 2 * NT; ++i)
                if (i < 2 * nvalid) raw[i >> 2] |= (int)((unsigned)q[i] << (8 * (i & 3)));
        }
    }
}

// out[2i], out[2i+1] = re, im of sample i as sign-extended ints.
template <int NT, bool I16>
__device__ __forceinline__ void unpack(const int *raw, int *out)
{
    if constexpr (I16) {
#pragma unroll
        for (int i = 0; i < NT; ++i) { out[2 * i] = (short)(raw[i] & 0xffff); out[2 * i + 1] = raw[i] >> 16; }
    } else {
#pragma unroll
        for (int i = 0; i < 2 * NT; ++i) out[i] = (signed char)((raw[i >> 2] >> (8 * (i & 3))) & 0xff);
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
    // Stations in groups of G: all 2*G row loads are issued before any of them is used.
    constexpr int NW = RowWords<NT, I16>::value;
    constexpr int G = (16 / NW) < 1 ? 1 : ((16 / NW) > 8 ? 8 : (16 / NW));
    for (int s0 = 0; s0 < a.S; s0 += G) {
        int raw[G][2][NW];
#pragma unroll
        for (int g = 0; g < G; ++g) {
            const int s = (s0 + g < a.S) ? s0 + g : a.S - 1;
            const char *r0 = Xb + ((size_t)(2 * s) * a.K + k) * row_bytes;
            load_raw<NT, I16>(r0, t, nvalid, raw[g][0]);
            load_raw<NT, I16>(r0 + (size_t)a.K * row_bytes, t, nvalid, raw[g][1]);
        }
#pragma unroll
        for (int g = 0; g < G; ++g) {
            if (s0 + g < a.S) {
                int v0[2 * NT], v1[2 * NT];
                unpack<NT, I16>(raw[g][0], v0);
                unpack<NT, I16>(raw[g][1], v1);
                float x[2 * NT];
#pragma unroll
                for (int i = 0; i < 2 * NT; ++i) x[i] = int_to_float_exact(v0[i] + v1[i]);
#pragma unroll
                for (int bb = 0; bb < BT; ++bb) {
                    const float2 w = sW[(s0 + g) * BT + bb];
#pragma unroll
                    for (int i = 0; i < NT; ++i) {
                        acc[bb][i].x = fmaf(w.x, x[2 * i], acc[bb][i].x);
                        acc[bb][i].x = fmaf(-w.y, x[2 * i + 1], acc[bb][i].x);
                        acc[bb][i].y = fmaf(w.x, x[2 * i + 1], acc[bb][i].y);
                        acc[bb][i].y = fmaf(w.y, x[2 * i], acc[bb][i].y);
                    }
                }
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
            float2 *zr = a.Z + (size_t)((b0 + bb) * nph + d) * a.K * (size_t)a.zpitch +
                         (a.ztile ? ((size_t)(col >> 4) * a.K + k) * 16 + (col & 15) : (size_t)k * a.zpitch + col);
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

// Two-stage beamforming: the first-stage beams leave as 16-bit integers.
// Z[g][k][q] float2 -> X2[g][pol 0][k][q] = clip(rint(Z * scale)) (ties to even), pol 1 = 0.
__global__ void __launch_bounds__(256) requantize_kernel(const float2 *Z, long long n_per_g, int G, float scale, short2 *X2)
{
    const long long i = (long long)blockIdx.x * 256 + threadIdx.x;
    const int g = blockIdx.y;
    if (i >= n_per_g) return;
    const float2 z = Z[(size_t)g * n_per_g + i];
    const int re = max(-32767, min(32767, __float2int_rn(z.x * scale)));
    const int im = max(-32767, min(32767, __float2int_rn(z.y * scale)));
    X2[(size_t)(2 * g) * n_per_g + i] = make_short2((short)re, (short)im);
    X2[(size_t)(2 * g + 1) * n_per_g + i] = make_short2(0, 0);
}

}  // namespace

int launch_requantize(const float2 *Z, long long n_per_g, int G, float scale, void *X2, cudaStream_t st)
{
    if (n_per_g <= 0) return 0;
    dim3 grid((unsigned)((n_per_g + 255) / 256), (unsigned)G);
    requantize_kernel<<<grid, 256, 0, st>>>(Z, n_per_g, G, scale, static_cast<short2 *>(X2));
    return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

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
