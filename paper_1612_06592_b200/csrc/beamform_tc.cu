// beamform_tc.cu -- step a1 on the 5th-generation tensor cores (tcgen05 + TMEM), int8 input.
//
// Per sub-band k the beam sum is a small real GEMM
//     D[t, n] = sum_kk A[t, kk] * Bw[n, kk],   t = 128 slices (M), kk = (station, re/im) (K = 2S),
//     n = (beam, re/im) (N = 2B),
// with A = the two polarisations added as integers (|sum| <= 256, exact in fp16) and Bw built from the
// weights: Bw[2b][2s] = Re W, Bw[2b][2s+1] = -Im W, Bw[2b+1][2s] = Im W, Bw[2b+1][2s+1] = Re W.
// fp16 weights alone (11 bits) would break the 1e-5 tolerance, so W = hi + lo with both halves fp16
// (22 bits) and two MMAs accumulate A*hi and A*lo into the same fp32 TMEM accumulator; every product
// is exact in fp32.  BASELINE.json:north_star makes this path conditional on the contraction being
// compute-bound at the largest beam count: profiles/r1_b shows the SIMT kernel at 70 % issue / 50 %
// FMA-pipe utilisation and 24 % of DRAM bandwidth for 24 beams.
//
// CTA = 128 threads, one sub-band, a run of 8 128-slice tiles.  Per tile: 96..128 threads each load
// 8 (station,pol) rows x 16 bytes, add the polarisations, convert to fp16 and write one 8x16-byte core
// matrix of the K-major no-swizzle operand layout; one thread issues the MMAs (kind::f16, M=128,
// N=2B padded to 16, K=16 per instruction) and commits to an mbarrier; the four warps read their 32
// TMEM lanes back with tcgen05.ld and store Z with 256-byte contiguous warp writes.
#include <cuda_fp16.h>

#include "plan.h"

namespace lofar {
namespace {

constexpr int kTcThreads = 128;
constexpr int kSboA = 144;              // bytes between 8-slice groups of A (128 + 16: conflict-free STS.128)
constexpr int kLboA = 16 * kSboA;       // bytes between K chunks (8 fp16) of A

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ uint64_t make_desc(uint32_t saddr, uint32_t lbo, uint32_t sbo)
{
    // K-major, SWIZZLE_NONE: [0,14) start>>4, [16,30) LBO>>4, [32,46) SBO>>4, [46,48) version = 1
    return (uint64_t)((saddr & 0x3FFFF) >> 4) | ((uint64_t)(lbo >> 4) << 16) | ((uint64_t)(sbo >> 4) << 32) |
           ((uint64_t)1 << 46);
}

__device__ __forceinline__ void mma_f16(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t acc)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}\n"
        :: "r"(tmem_d), "l"(da), "l"(db), "r"(idesc), "r"(acc) : "memory");
}

__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    asm volatile(
        "{\n\t.reg .pred P1;\n\tLAB_WAIT:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n\t"
        "@P1 bra DONE;\n\tbra LAB_WAIT;\n\tDONE:\n\t}\n"
        :: "r"(bar), "r"(parity) : "memory");
}

// (int8 ^ 0x80) placed under the fp16 exponent 0x64 reads as 1152 + v; subtracting 1152 is exact.
__device__ __forceinline__ __half2 bytes_to_half2(uint32_t word_xor, uint32_t sel)
{
    uint32_t h = __byte_perm(word_xor, 0x64646464u, sel);
    __half2 r = *reinterpret_cast<__half2 *>(&h);
    return __hsub2(r, __float2half2_rn(1152.0f));
}

struct TcArgs {
    BeamformArgs b;
    const uint4 *wimg;     // [K][2][img16] operand images of Bw (hi, lo)
    int img16;             // uint4 per image
    int kchunks;           // K chunks of 8 fp16 (2 per MMA)
    int np;                // padded N
    int tiles_per_cta;
};

__global__ void __launch_bounds__(kTcThreads) beamform_tc_kernel(TcArgs a)
{
    extern __shared__ __align__(128) unsigned char smem[];
    // layout: [A: kchunks*kLboA][Bhi: img][Blo: img][mbar 8][tmem ptr 4]
    unsigned char *sA = smem;
    const int a_bytes = a.kchunks * kLboA;
    uint4 *sB = reinterpret_cast<uint4 *>(smem + a_bytes);
    const int b_bytes = a.img16 * 16;
    uint64_t *mbar = reinterpret_cast<uint64_t *>(smem + a_bytes + 2 * b_bytes);
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(mbar + 1);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int k = blockIdx.x;           // sub-band fastest: CTAs running together write neighbouring lines of a Z tile
    const BeamformArgs &g = a.b;

    // weights image of this sub-band, zero the A tile once (pad stations stay zero)
    const uint4 *src = a.wimg + (size_t)k * 2 * a.img16;
    for (int i = tid; i < 2 * a.img16; i += kTcThreads) sB[i] = src[i];
    for (int i = tid; i < a_bytes / 16; i += kTcThreads) reinterpret_cast<uint4 *>(sA)[i] = make_uint4(0, 0, 0, 0);
    if (tid == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" :: "r"(smem_u32(mbar)));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    uint32_t ncols = 32;
    while ((int)ncols < a.np) ncols <<= 1;
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;"
                     :: "r"(smem_u32(tmem_slot)), "r"(ncols) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem = *tmem_slot;

    // unit of this thread: K chunk c (stations 4c..4c+3), slice group grp (8 slices)
    const int grp = tid & 15, c = tid >> 4;
    const bool loader = c < a.kchunks;
    const size_t row_bytes = (size_t)g.xpitch * 2;
    const char *Xb = reinterpret_cast<const char *>(g.X);
    const uint32_t idesc = (1u << 4) | ((uint32_t)(a.np >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
    const uint32_t sA_addr = smem_u32(sA), sB_addr = smem_u32(sB);
    const uint32_t lbo_b = (uint32_t)(a.np / 8) * 128;

    const long long tile0 = (long long)blockIdx.y * a.tiles_per_cta;
    uint32_t phase = 0;
    for (int it = 0; it < a.tiles_per_cta; ++it) {
        const long long col0 = (tile0 + it) * 128;       // column in Z / offset inside this launch
        if (col0 >= g.nt) break;
        // ---- operand A: load, add polarisations, convert, store one core matrix per thread ----
        if (loader) {
            const long long col = col0 + grp * 8;
            uint4 raw[4][2];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int s = 4 * c + j;
                const bool ok = s < g.S && col < g.nt;      // rows are whole 16-byte groups (pitch % 8 == 0)
#pragma unroll
                for (int p = 0; p < 2; ++p) {
                    raw[j][p] = make_uint4(0x80808080u, 0x80808080u, 0x80808080u, 0x80808080u) ;
                    if (ok) {
                        const char *r = Xb + ((size_t)(2 * s + p) * g.K + k) * row_bytes + (size_t)(g.t0 + col) * 2;
                        const uint4 v = __ldg(reinterpret_cast<const uint4 *>(r));
                        raw[j][p] = make_uint4(v.x ^ 0x80808080u, v.y ^ 0x80808080u, v.z ^ 0x80808080u, v.w ^ 0x80808080u);
                    }
                }
            }
            // slices beyond nt inside a 16-byte group cannot occur for loads (nt is a multiple of 8 or the
            // row ends there); their outputs are masked at the store.
            unsigned char *dst = sA + c * kLboA + grp * kSboA;
#pragma unroll
            for (int w = 0; w < 4; ++w) {                  // word w holds slices 2w, 2w+1
                __half2 lo2[4], hi2[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const uint32_t x0 = (&raw[j][0].x)[w], x1 = (&raw[j][1].x)[w];
                    lo2[j] = __hadd2(bytes_to_half2(x0, 0x4140), bytes_to_half2(x1, 0x4140));   // slice 2w: bytes 0,1
                    hi2[j] = __hadd2(bytes_to_half2(x0, 0x4342), bytes_to_half2(x1, 0x4342));   // slice 2w+1: bytes 2,3
                }
                uint4 o0, o1;
                o0.x = *reinterpret_cast<uint32_t *>(&lo2[0]); o0.y = *reinterpret_cast<uint32_t *>(&lo2[1]);
                o0.z = *reinterpret_cast<uint32_t *>(&lo2[2]); o0.w = *reinterpret_cast<uint32_t *>(&lo2[3]);
                o1.x = *reinterpret_cast<uint32_t *>(&hi2[0]); o1.y = *reinterpret_cast<uint32_t *>(&hi2[1]);
                o1.z = *reinterpret_cast<uint32_t *>(&hi2[2]); o1.w = *reinterpret_cast<uint32_t *>(&hi2[3]);
                *reinterpret_cast<uint4 *>(dst + (2 * w) * 16) = o0;
                *reinterpret_cast<uint4 *>(dst + (2 * w + 1) * 16) = o1;
            }
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();
        // ---- MMA: D = A * Bhi^T + A * Blo^T ----
        if (tid == 0) {
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            uint32_t acc = 0;
            for (int half = 0; half < 2; ++half) {
                for (int ks = 0; ks < a.kchunks / 2; ++ks) {
                    const uint64_t da = make_desc(sA_addr + (uint32_t)ks * 2 * kLboA, kLboA, kSboA);
                    const uint64_t db = make_desc(sB_addr + (uint32_t)half * b_bytes + (uint32_t)ks * 2 * lbo_b, lbo_b, 128);
                    mma_f16(tmem, da, db, idesc, acc);
                    acc = 1;
                }
            }
            asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];"
                         :: "r"(smem_u32(mbar)) : "memory");
        }
        mbar_wait(smem_u32(mbar), phase);
        phase ^= 1;
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        // ---- epilogue: thread = slice col0 + 32*warp + lane, 16 accumulator columns (8 beams) at a time ----
        const long long colt = col0 + warp * 32 + lane;
        for (int n0 = 0; n0 < a.np; n0 += 16) {
            uint32_t r[16];
            const uint32_t taddr = tmem + ((uint32_t)(warp * 32) << 16) + (uint32_t)n0;
            asm volatile(
                "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];\n\t"
                "tcgen05.wait::ld.sync.aligned;"
                : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
                  "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
                : "r"(taddr) : "memory");
            if (colt < g.nt) {
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    const int b = n0 / 2 + j;
                    if (b < g.B) {
                        float2 *zr = g.Z + (size_t)b * g.K * (size_t)g.zpitch +
                                     (g.ztile ? ((size_t)(colt >> 4) * g.K + k) * 16 + (colt & 15)
                                              : (size_t)k * g.zpitch + colt);
                        *zr = make_float2(__uint_as_float(r[2 * j]), __uint_as_float(r[2 * j + 1]));
                    }
                }
            }
        }
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();     // TMEM drained and A consumed before the next tile overwrites them
    }

    if (warp == 0) {
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(tmem), "r"(ncols) : "memory");
    }
}

}  // namespace

// Host: operand image of Bw for one sub-band and one half (hi or lo), K-major no-swizzle core matrices:
// element (n, kk) at byte (kk/8)*lbo + (n/8)*128 + (n%8)*16 + (kk%8)*2 with lbo = (np/8)*128.
size_t tc_image_halfs(int S, int B)
{
    const int kp = (2 * S + 15) / 16 * 16, np = (2 * B + 15) / 16 * 16;
    return (size_t)kp * np;
}

void tc_build_image(const double *w_re, const double *w_im, int S, int B, unsigned short *hi, unsigned short *lo)
{
    const int kp = (2 * S + 15) / 16 * 16, np = (2 * B + 15) / 16 * 16;
    const size_t lbo = (size_t)(np / 8) * 128;
    for (size_t i = 0; i < (size_t)kp * np; ++i) hi[i] = lo[i] = 0;
    for (int b = 0; b < B; ++b)
        for (int s = 0; s < S; ++s) {
            const double re = w_re[b * S + s], im = w_im[b * S + s];
            const double v[2][2] = {{re, -im}, {im, re}};     // [c' (out re/im)][c (in re/im)]
            for (int co = 0; co < 2; ++co)
                for (int ci = 0; ci < 2; ++ci) {
                    const int n = 2 * b + co, kk = 2 * s + ci;
                    const size_t byte = (size_t)(kk / 8) * lbo + (size_t)(n / 8) * 128 + (size_t)(n % 8) * 16 + (size_t)(kk % 8) * 2;
                    const __half h = __float2half_rn((float)v[co][ci]);
                    const __half l = __float2half_rn((float)(v[co][ci] - (double)__half2float(h)));
                    hi[byte / 2] = *reinterpret_cast<const unsigned short *>(&h);
                    lo[byte / 2] = *reinterpret_cast<const unsigned short *>(&l);
                }
        }
}

bool tc_supported(const BeamformArgs &a)
{
    return a.dtype == LOFAR_CI8 && a.nphase == 0 && a.S <= 32 && a.B <= 128 && (a.xpitch % 8) == 0 &&
           (a.t0 % 8) == 0;
}

// Per device (function attributes are per context): called from every plan build, result checked there.
int tc_configure()
{
    cudaError_t e = cudaFuncSetAttribute(beamform_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    return e == cudaSuccess ? 0 : -1;
}

int launch_beamform_tc(const BeamformArgs &b, const void *wimg, cudaStream_t st)
{
    if (b.nt <= 0) return 0;
    TcArgs a;
    a.b = b;
    const int kp = (2 * b.S + 15) / 16 * 16;
    a.np = (2 * b.B + 15) / 16 * 16;
    a.kchunks = kp / 8;
    a.img16 = (int)(tc_image_halfs(b.S, b.B) * 2 / 16);
    a.wimg = static_cast<const uint4 *>(wimg);
    const long long tiles = (b.nt + 127) / 128;
    // 8 tiles (1024 slices) per CTA: measured optimum on B200 for configs[2] (ms per block for 1 / 2 / 4 / 8 / 16 / 32 / 88
    // tiles: 5.09 / 3.68 / 3.30 / 3.22 / 3.34 / 3.45 / 3.81) -- long enough to amortise the per-CTA prologue (weight
    // images, TMEM allocation), short enough that the CTAs in flight write a narrow band of Z tiles
#ifndef LOFAR_BF_TILES
#define LOFAR_BF_TILES 8
#endif
    a.tiles_per_cta = tiles < LOFAR_BF_TILES ? (int)tiles : LOFAR_BF_TILES;
    dim3 grid((unsigned)b.K, (unsigned)((tiles + a.tiles_per_cta - 1) / a.tiles_per_cta));
    const size_t smem = (size_t)a.kchunks * kLboA + 2 * (size_t)a.img16 * 16 + 16;
    beamform_tc_kernel<<<grid, kTcThreads, smem, st>>>(a);
    return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

}  // namespace lofar
