// fft_warp.cuh -- packed fp32x2 arithmetic and the warp-level 512-point inverse complex FFT shared by the
// inverse polyphase filter (ippf.cu, step a3) and the exact de-dispersion (dedisp.cu, row f2).
// Device code only; nothing here is shared with oracle/.
#pragma once
#include "fft_math.cuh"

namespace lofar {

typedef unsigned long long u64;

// ---- packed fp32x2 helpers: a u64 is an aligned register pair (lo = .x, hi = .y) -------------------
__device__ __forceinline__ u64 PK(float x, float y) { u64 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(x), "f"(y)); return r; }
__device__ __forceinline__ float LO(u64 v) { float x; asm("{\n\t.reg .f32 t;\n\tmov.b64 {%0, t}, %1;\n\t}" : "=f"(x) : "l"(v)); return x; }
__device__ __forceinline__ float HI(u64 v) { float y; asm("{\n\t.reg .f32 t;\n\tmov.b64 {t, %0}, %1;\n\t}" : "=f"(y) : "l"(v)); return y; }
// fma2p is always the packed instruction; add2 / sub2 / fma2 are the transform's arithmetic and
// become scalar pairs with -DLOFAR_FFT_SCALAR (ablation: packed instructions with distinct register operands are
// register-file limited to ~79 FMA/clk/SM against ~100 for scalar ones, but take half the issue slots).
__device__ __forceinline__ u64 fma2p(u64 a, u64 b, u64 c) { u64 d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d; }
#ifdef LOFAR_FFT_SCALAR
__device__ __forceinline__ u64 add2(u64 a, u64 b) { return PK(LO(a) + LO(b), HI(a) + HI(b)); }
__device__ __forceinline__ u64 sub2(u64 a, u64 b) { return PK(LO(a) - LO(b), HI(a) - HI(b)); }
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c) { return PK(fmaf(LO(a), LO(b), LO(c)), fmaf(HI(a), HI(b), HI(c))); }
#else
__device__ __forceinline__ u64 add2(u64 a, u64 b) { u64 d; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ u64 sub2(u64 a, u64 b) { u64 d; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c) { return fma2p(a, b, c); }
#endif
__device__ __forceinline__ u64 lds64(const float2 *p) { return *reinterpret_cast<const u64 *>(p); }
__device__ __forceinline__ void sts64(float2 *p, u64 v) { *reinterpret_cast<u64 *>(p) = v; }
// a * (c + i s), scalar products (a complex product needs the swapped pair, which the packed forms lack)
__device__ __forceinline__ u64 cmulp(u64 a, float c, float s)
{
    const float ax = LO(a), ay = HI(a);
    return PK(fmaf(c, ax, -s * ay), fmaf(c, ay, s * ax));
}
// a + i b and a - i b
__device__ __forceinline__ u64 addi(u64 a, u64 b) { return PK(LO(a) - HI(b), HI(a) + LO(b)); }
__device__ __forceinline__ u64 subi(u64 a, u64 b) { return PK(LO(a) + HI(b), HI(a) - LO(b)); }

// Inverse 8-point DFT in place on packed complex values: x[m] <- sum_r x[r] exp(+2 pi i r m / 8).
__device__ __forceinline__ void idft8p(u64 *x)
{
    const float s = 0.70710678118654752440f;
    const u64 a0 = add2(x[0], x[4]), a1 = sub2(x[0], x[4]);
    const u64 a2 = add2(x[2], x[6]), a3 = sub2(x[2], x[6]);
    const u64 e0 = add2(a0, a2), e2 = sub2(a0, a2), e1 = addi(a1, a3), e3 = subi(a1, a3);
    const u64 b0 = add2(x[1], x[5]), b1 = sub2(x[1], x[5]);
    const u64 b2 = add2(x[3], x[7]), b3 = sub2(x[3], x[7]);
    const u64 o0 = add2(b0, b2), o2 = sub2(b0, b2), o1 = addi(b1, b3), o3 = subi(b1, b3);
    // odd part times W8^m = exp(+i pi m / 4):  o1 (1+i)/sqrt2 = s (x - y, x + y);  o3 (-1+i)/sqrt2 = s (-(x + y), x - y)
    const u64 q1 = PK(LO(o1) - HI(o1), LO(o1) + HI(o1));
    const u64 q3 = PK(LO(o3) + HI(o3), LO(o3) - HI(o3));
    x[0] = add2(e0, o0); x[4] = sub2(e0, o0);
    x[1] = fma2(q1, PK(s, s), e1); x[5] = fma2(q1, PK(-s, -s), e1);
    x[2] = addi(e2, o2); x[6] = subi(e2, o2);
    x[3] = fma2(q3, PK(-s, s), e3); x[7] = fma2(q3, PK(s, -s), e3);
}

// Inverse 16-point DFT in place (two 8-point DFTs of the even / odd inputs, then the W16^m butterflies).
__device__ __forceinline__ void idft16p(u64 *x)
{
    u64 e[8], o[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) { e[i] = x[2 * i]; o[i] = x[2 * i + 1]; }
    idft8p(e);
    idft8p(o);
    const float c1 = 0.92387953251128675613f, s1 = 0.38268343236508977173f, h = 0.70710678118654752440f;
    x[0] = add2(e[0], o[0]); x[8] = sub2(e[0], o[0]);
    { const u64 t = cmulp(o[1], c1, s1); x[1] = add2(e[1], t); x[9] = sub2(e[1], t); }
    { const u64 q = PK(LO(o[2]) - HI(o[2]), LO(o[2]) + HI(o[2])); x[2] = fma2(q, PK(h, h), e[2]); x[10] = fma2(q, PK(-h, -h), e[2]); }
    { const u64 t = cmulp(o[3], s1, c1); x[3] = add2(e[3], t); x[11] = sub2(e[3], t); }
    x[4] = addi(e[4], o[4]); x[12] = subi(e[4], o[4]);
    { const u64 t = cmulp(o[5], -s1, c1); x[5] = add2(e[5], t); x[13] = sub2(e[5], t); }
    { const u64 q = PK(LO(o[6]) + HI(o[6]), LO(o[6]) - HI(o[6])); x[6] = fma2(q, PK(-h, h), e[6]); x[14] = fma2(q, PK(h, -h), e[6]); }
    { const u64 t = cmulp(o[7], -c1, s1); x[7] = add2(e[7], t); x[15] = sub2(e[7], t); }
}

// Radix-32 pass of the 512-point inverse FFT (512 = 16 x 32) of one slice row by one warp, in place. The row holds
// the radix-16 results at 16 j + m. Butterfly j (0..15) is a 32-point DFT of elements j + 16 r with twiddles
// TB[r][j] = exp(2 pi i j r / 512) (TW: applied here on load; otherwise the producer of the row has applied them);
// lanes j and j + 16 share it: the low lane does the 16-point DFT E of the even r, the high lane that of the odd r, O.
// The table carries a factor (-1)^((r-1)/2) on its odd rows (TBs, built in api.cu): the inputs of the high lane
// arrive as (-1)^r' x[r'], which rotates its outputs by 8 -- register i holds O[(i + 8) mod 16] -- so that both
// lanes can hand over the SAME registers 8..15 (E[8..15] one way, W32^i O[i] the other) in 8 exchanges instead of 16:
// the low lane finishes outputs i and 16 + i, the high lane 8 + i and 24 + i (i < 8); output m goes to j + 16 m.
template <bool TW>
__device__ __forceinline__ void fft512_pass_b(float2 *row, const float2 *stw, int lane)
{
    u64 x[16];
    // pad(lane + 32 r) = lane + (lane >> 4) + 34 r: one base pointer and compile-time offsets
    const float2 *src = row + lane + (lane >> 4);
    if (TW) {
        const float2 *T = stw + 256 + lane;      // T[32 r' + lane] = TBs[2 r' + hh][lane & 15]
#pragma unroll
        for (int r = 0; r < 16; ++r) {
            const float2 t = T[32 * r];
            x[r] = cmulp(lds64(src + 34 * r), t.x, t.y);
        }
    } else {
#pragma unroll
        for (int r = 0; r < 16; ++r) x[r] = lds64(src + 34 * r);
    }
    idft16p(x);
    const bool hi = lane >= 16;
    if (hi) {
        // register i holds O[k], k = (i + 8) mod 16: times W32^k = exp(2 pi i k / 32)
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
        for (int i = 0; i < 16; ++i) {
            const int k = (i + 8) & 15;
            if (k) x[i] = cmulp(x[i], c[k], sn[k]);
        }
    }
    // low lane: own = E[i], received = W32^i O[i]; high lane: own = W32^(8+i) O[8+i], received = E[8+i]
    const u64 sg = hi ? PK(-1.f, -1.f) : PK(1.f, 1.f);
    __syncwarp();
    const int jl = lane & 15;
    float2 *dsum = row + jl + (hi ? 17 * 8 : 0);               // outputs i (low) / 8 + i (high): pad(j + 16 m) = j + 17 m
    float2 *ddif = row + jl + (hi ? 17 * 24 : 17 * 16);        // outputs 16 + i (low) / 24 + i (high)
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const u64 other = __shfl_xor_sync(0xffffffffu, x[8 + i], 16);
        const u64 s2 = add2(x[i], other);                      // E + W O on either lane
        const u64 d2 = sub2(x[i], other);                      // low: E - W O;  high: W O - E
        x[i] = s2;
        x[8 + i] = fma2(d2, sg, 0ull);
    }
    __syncwarp();
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        sts64(dsum + 17 * i, x[i]);
        sts64(ddif + 17 * i, x[8 + i]);
    }
    __syncwarp();
}

// 512-point inverse complex FFT of one slice row by one warp, in place:
//   pass A: lane j does the 16-point DFT of elements j + 32 r and writes them to 16 j + m;
//   pass B: fft512_pass_b with the twiddles applied on load.
__device__ __forceinline__ void fft512_warp(float2 *row, const float2 *stw, int lane)
{
    u64 x[16];
    const float2 *src = row + lane + (lane >> 4);          // pad(lane + 32 r) = lane + (lane >> 4) + 34 r
#pragma unroll
    for (int r = 0; r < 16; ++r) x[r] = lds64(src + 34 * r);
    idft16p(x);
    __syncwarp();
    float2 *dst = row + 17 * lane;                         // pad(16 lane + m) = 17 lane + m
#pragma unroll
    for (int m = 0; m < 16; ++m) sts64(dst + m, x[m]);
    __syncwarp();
    fft512_pass_b<true>(row, stw, lane);
}

}  // namespace lofar
