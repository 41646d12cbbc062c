// lsmr.cu -- row f1 of SURVEY.md 8(f): least-squares inversion of the polyphase filter by LSMR
// (section 3: "a system of sparse linear equations H x^ = y where H is the matrix of the FIR
// filters ... solved by an iterative LSMR algorithm [14] ... convergence ... after approximately 25 iterations";
// Fong & Saunders; reading A23 in DESIGN.md).
//
// H is block diagonal over the 1024 residues: residue r of one series is its own banded system
//     (A v)[m]   = sum_{t<16} taps[t][r] v[m + t],   m = 0 .. n_eq-1   (n_eq = 15 carried + T slices of y)
//     (A^T u)[n] = sum_{t<16} taps[t][r] u[n - t],   n = 0 .. n_un-1   (n_un = n_eq + 15 unknown slices)
// with b = y / 1024.  Every (series, residue) runs the LSMR recurrences with its own scalars; nothing couples
// them, so the vectors are laid out [row][1024] and a thread owns one residue of a run of rows: loads are
// coalesced over residues and the 16-tap window slides through registers along the rows, 8 rows at a time with all
// loads of a group issued before its arithmetic (the solver is a stream of 13 vector passes per iteration).
// Vectors are kept unnormalised (u', v') next to their norms (beta, alpha): a pass never has to wait for a norm
// it produces itself.  Norms: per-chunk partial sums in double, added in a fixed order.
#include "plan.h"

namespace lofar {
namespace {

constexpr int kTapsN = 16, kRes = 1024, kRows = 64;      // rows per CTA
constexpr int kLsmrThreads = 256;
#ifndef LOFAR_LSMR_G
#define LOFAR_LSMR_G 8
#endif
#ifndef LOFAR_U_MINB
#define LOFAR_U_MINB 4
#endif
#ifndef LOFAR_UH_MINB
#define LOFAR_UH_MINB 2
#endif
#ifndef LOFAR_V_MINB
#define LOFAR_V_MINB 4
#endif
constexpr int kG = LOFAR_LSMR_G;           // rows per group: their loads are issued together

// Scalars of one (series, residue), double precision (Fong & Saunders, "Algorithm LSMR", lambda = 0).
struct Scal {
    double alpha, beta, alphabar, zetabar, rho, rhobar, cbar, sbar;
    double inv_alpha, inv_beta;          // 1/alpha, 1/beta of the stored (unnormalised) v', u'
    double ch, cx, cv;                   // hbar = h - ch hbar; x += cx hbar; h = v - cv h
    double cxp;                          // cx of the previous iteration (its x update may still be pending)
};

__device__ __forceinline__ double safe_div(double a, double d) { return d != 0.0 ? a / d : 0.0; }

// u'[m] = sum_t taps[t] v'[m+t] / alpha - alpha * u'[m] / beta_old    (first = 0)
// or first = 1:  u' = b / 1024 (the right-hand side), nothing else.
// Groups of 8 rows and 4 CTAs per SM for both kernels: measured optimum on B200 (ms per configs[2] block of 25 iterations,
// group / CTAs of u / CTAs of v: 16/1/1 872, 16/4/3 705, 8/4/4 672, 8/5/4 783, 8/6/5 1009, 4/4/4 716, 12/4/4 695, 32/2/2 845)
// HM >= 0: the h / hbar / x update of the PREVIOUS iteration (h_kernel with xmode = HM) is done here for rows 0 .. n_eq-1,
// on the v' values this kernel holds in its window anyway -- v' is then read once per iteration instead of twice; the
// last 15 rows (n_eq .. n_un-1) are left to a small h_kernel launch.  h, hbar, x share the pitch of v'.
template <int HM>
__global__ void __launch_bounds__(kLsmrThreads, HM >= 0 ? LOFAR_UH_MINB : LOFAR_U_MINB)
u_kernel(float *u, long long upitch, long long n_eq, const float *v, long long vpitch, const float *gs, const Scal *sc,
         double *partial, int nchunks, int first, float *h, float *hbar, float *x)
{
    const int r = blockIdx.x * kLsmrThreads + threadIdx.x, chunk = blockIdx.y, series = blockIdx.z;
    float *pu = u + (size_t)series * upitch + r;
    const long long m0 = (long long)chunk * kRows, m1 = m0 + kRows < n_eq ? m0 + kRows : n_eq;
    double s = 0.0;
    if (first) {
        for (long long m = m0; m < m1; ++m) {
            const float val = pu[(size_t)m * kRes] * (1.0f / 1024.0f);
            pu[(size_t)m * kRes] = val;
            s += (double)val * val;
        }
    } else {
        const Scal z = sc[(size_t)series * kRes + r];
        const float ia = (float)z.inv_alpha, ab = (float)(z.alpha * z.inv_beta);
        const float *pv = v + (size_t)series * vpitch + r;
        // rows in groups of 16: the 16 new rows of v' and the 16 rows of u' are loaded before anything is computed (32
        // independent loads per thread in flight -- the kernel is a stream and lives on memory-level parallelism); the
        // window w[0..30] = v'[mb .. mb+30] slides by 16 registers per group
        float tap[kTapsN], w[kTapsN - 1 + kG];
#pragma unroll
        for (int t = 0; t < kTapsN; ++t) tap[t] = gs[t * kRes + r] * (1.0f / 1024.0f);
#pragma unroll
        for (int t = 0; t < kTapsN - 1; ++t) w[t] = pv[(size_t)(m0 + t) * kRes];
        const float ch = (float)z.ch, cx = (float)z.cx, cv = (float)z.cv, cxp = (float)z.cxp;
        const size_t hbase = (size_t)series * vpitch + r;
        for (long long mb = m0; mb < m1; mb += kG) {
            float un[kG], hh[HM >= 0 ? kG : 1], hb[HM >= 0 ? kG : 1], xx[(HM == 0 || HM == 2) ? kG : 1];
#pragma unroll
            for (int k = 0; k < kG; ++k) {
                const bool ok = mb + k < m1;                     // rows m .. m+15 of v' exist for m < n_eq (n_un = n_eq + 15)
                w[kTapsN - 1 + k] = ok ? pv[(size_t)(mb + k + kTapsN - 1) * kRes] : 0.f;
                un[k] = ok ? pu[(size_t)(mb + k) * kRes] : 0.f;
                if (HM >= 0) {
                    const size_t i = hbase + (size_t)(mb + k) * kRes;
                    hh[k] = ok ? h[i] : 0.f;
                    hb[k] = ok ? hbar[i] : 0.f;
                    if (HM == 0 || HM == 2) xx[k] = ok ? x[i] : 0.f;
                }
            }
            if (HM >= 0) {
#pragma unroll
                for (int k = 0; k < kG; ++k) {
                    if (mb + k < m1) {
                        const size_t i = hbase + (size_t)(mb + k) * kRes;
                        const float vn = w[k] * ia;              // v' of row mb + k
                        const float b = fmaf(-ch, hb[k], hh[k]);
                        hbar[i] = b;
                        if (HM == 0) x[i] = fmaf(cx, b, xx[k]);
                        if (HM == 2) x[i] = fmaf(cx, b, fmaf(cxp, hb[k], xx[k]));
                        h[i] = fmaf(-cv, hh[k], vn);
                    }
                }
            }
#pragma unroll
            for (int k = 0; k < kG; ++k) {
                float acc = 0.f;
#pragma unroll
                for (int t = 0; t < kTapsN; ++t) acc = fmaf(tap[t], w[k + t], acc);
                const float val = fmaf(acc, ia, -ab * un[k]);
                if (mb + k < m1) {
                    pu[(size_t)(mb + k) * kRes] = val;
                    s += (double)val * val;
                }
            }
#pragma unroll
            for (int t = 0; t < kTapsN - 1; ++t) w[t] = w[t + kG];
        }
    }
    partial[((size_t)series * nchunks + chunk) * kRes + r] = s;
}

// v'[n] = sum_t taps[t] u'[n-t] / beta - beta * v'[n] / alpha_old     (first: no second term)
__global__ void __launch_bounds__(kLsmrThreads, LOFAR_V_MINB) v_kernel(float *v, long long vpitch, long long n_un, const float *u,
                                                         long long upitch, long long n_eq, const float *gs, const Scal *sc,
                                                         double *partial, int nchunks, int first)
{
    const int r = blockIdx.x * kLsmrThreads + threadIdx.x, chunk = blockIdx.y, series = blockIdx.z;
    float *pv = v + (size_t)series * vpitch + r;
    const float *pu = u + (size_t)series * upitch + r;
    const long long n0 = (long long)chunk * kRows, n1 = n0 + kRows < n_un ? n0 + kRows : n_un;
    const Scal z = sc[(size_t)series * kRes + r];
    const float ib = (float)z.inv_beta, ba = first ? 0.f : (float)(z.beta * z.inv_alpha);
    // as u_kernel: groups of 16 rows, loads first. w[j] = u'[nb - 15 + j], j = 0..30 (zero outside 0 .. n_eq-1)
    float tap[kTapsN], w[kTapsN - 1 + kG];
#pragma unroll
    for (int t = 0; t < kTapsN; ++t) tap[t] = gs[t * kRes + r] * (1.0f / 1024.0f);
#pragma unroll
    for (int j = 0; j < kTapsN - 1; ++j) {
        const long long m = n0 - (kTapsN - 1) + j;
        w[j] = (m >= 0 && m < n_eq) ? pu[(size_t)m * kRes] : 0.f;
    }
    double s = 0.0;
    for (long long nb = n0; nb < n1; nb += kG) {
        float vo[kG];
#pragma unroll
        for (int k = 0; k < kG; ++k) {
            const long long n = nb + k;
            w[kTapsN - 1 + k] = (n < n1 && n < n_eq) ? pu[(size_t)n * kRes] : 0.f;
            vo[k] = (!first && n < n1) ? pv[(size_t)n * kRes] : 0.f;
        }
#pragma unroll
        for (int k = 0; k < kG; ++k) {
            float acc = 0.f;
#pragma unroll
            for (int t = 0; t < kTapsN; ++t) acc = fmaf(tap[t], w[kTapsN - 1 + k - t], acc);    // u'[n - t]
            float val = acc * ib;
            if (!first) val = fmaf(-ba, vo[k], val);
            if (nb + k < n1) {
                pv[(size_t)(nb + k) * kRes] = val;
                s += (double)val * val;
            }
        }
#pragma unroll
        for (int j = 0; j < kTapsN - 1; ++j) w[j] = w[j + kG];
    }
    partial[((size_t)series * nchunks + chunk) * kRes + r] = s;
}

// which: 0 beta_1 (start), 1 alpha_1 + initial scalars, 2 beta_{k+1}, 3 alpha_{k+1} + the plane rotations.
__global__ void __launch_bounds__(kLsmrThreads) scalar_kernel(Scal *sc, const double *partial, int nchunks, int which)
{
    const int r = blockIdx.x * kLsmrThreads + threadIdx.x, series = blockIdx.y;
    const double *p = partial + (size_t)series * nchunks * kRes + r;
    double s = 0.0;
    for (int c = 0; c < nchunks; ++c) s += p[(size_t)c * kRes];
    const double nrm = sqrt(s);
    Scal z = sc[(size_t)series * kRes + r];
    if (which == 0) {
        z.beta = nrm; z.inv_beta = safe_div(1.0, nrm);
    } else if (which == 1) {
        z.alpha = nrm; z.inv_alpha = safe_div(1.0, nrm);
        z.alphabar = z.alpha; z.zetabar = z.alpha * z.beta;
        z.rho = 1.0; z.rhobar = 1.0; z.cbar = 1.0; z.sbar = 0.0;
        z.ch = 0.0; z.cx = 0.0; z.cv = 0.0; z.cxp = 0.0;
    } else if (which == 2) {
        z.beta = nrm; z.inv_beta = safe_div(1.0, nrm);
    } else {
        z.alpha = nrm; z.inv_alpha = safe_div(1.0, nrm);
        const double rhoold = z.rho;
        z.rho = hypot(z.alphabar, z.beta);
        const double c = safe_div(z.alphabar, z.rho), s1 = safe_div(z.beta, z.rho);
        const double thetanew = s1 * z.alpha;
        z.alphabar = c * z.alpha;
        const double rhobarold = z.rhobar;
        const double thetabar = z.sbar * z.rho;
        const double rhotemp = z.cbar * z.rho;
        z.rhobar = hypot(rhotemp, thetanew);
        z.cbar = safe_div(rhotemp, z.rhobar);
        z.sbar = safe_div(thetanew, z.rhobar);
        const double zeta = z.cbar * z.zetabar;
        z.zetabar = -z.sbar * z.zetabar;
        z.cxp = z.cx;
        z.ch = safe_div(thetabar * z.rho, rhoold * rhobarold);
        z.cx = safe_div(zeta, z.rho * z.rhobar);
        z.cv = safe_div(thetanew, z.rho);
    }
    sc[(size_t)series * kRes + r] = z;
}

// first: h = v'/alpha, hbar = 0, x = 0.   else: hbar = h - ch hbar; x += cx hbar; h = v'/alpha - cv h.
// xmode (x is only needed after the last iteration, so its update is applied every other iteration and x makes one
// round trip through HBM instead of two): 0 = this iteration's term now; 1 = defer it (x untouched); 2 = the deferred
// term of the previous iteration, cxp * hbar_old, then this one -- the same two fused multiply-adds in the same order
// as two separate updates, so the result is bit-identical.
__global__ void __launch_bounds__(kLsmrThreads) h_kernel(float *h, float *hbar, float *x, const float *v, long long pitch,
                                                         long long n_un, const Scal *sc, int first, int xmode,
                                                         float *series, long long series_pitch, long long T, long long n_begin)
{
    // series != nullptr (the last iteration): the solution leaves through here -- series[q][r] = x[q + 15][r] -- instead
    // of going back to the work vector and through a copy kernel
    const int r = blockIdx.x * kLsmrThreads + threadIdx.x, chunk = blockIdx.y, series_idx = blockIdx.z;
    const Scal z = sc[(size_t)series_idx * kRes + r];
    const float ia = (float)z.inv_alpha, ch = (float)z.ch, cx = (float)z.cx, cv = (float)z.cv, cxp = (float)z.cxp;
    const size_t base = (size_t)series_idx * pitch + r;
    const long long n0 = n_begin + (long long)chunk * kRows, n1 = n0 + kRows < n_un ? n0 + kRows : n_un;
    for (long long nb = n0; nb < n1; nb += 4) {
        float vv[4], hh[4], hb[4], xx[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {                 // loads of four rows first (memory-level parallelism)
            const bool ok = nb + k < n1;
            const size_t i = base + (size_t)(nb + k) * kRes;
            vv[k] = ok ? v[i] : 0.f;
            if (!first) {
                hh[k] = ok ? h[i] : 0.f; hb[k] = ok ? hbar[i] : 0.f;
                xx[k] = (ok && xmode != 1) ? x[i] : 0.f;
            }
        }
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            if (nb + k >= n1) break;
            const size_t i = base + (size_t)(nb + k) * kRes;
            const float vn = vv[k] * ia;
            if (first) { h[i] = vn; hbar[i] = 0.f; x[i] = 0.f; }
            else {
                const float b = fmaf(-ch, hb[k], hh[k]);
                hbar[i] = b;
                if (xmode != 1) {
                    const float xn = fmaf(cx, b, xmode == 2 ? fmaf(cxp, hb[k], xx[k]) : xx[k]);
                    if (series) {
                        const long long q = nb + k - (kTapsN - 1);
                        if (q >= 0 && q < T) series[(size_t)series_idx * series_pitch + (size_t)q * kRes + r] = xn;
                    } else x[i] = xn;
                }
                h[i] = fmaf(-cv, hh[k], vn);
            }
        }
    }
}

}  // namespace

size_t lsmr_scalar_bytes(int nseries) { return (size_t)nseries * kRes * sizeof(Scal); }
size_t lsmr_partial_count(int nseries, long long n_un) { return (size_t)nseries * ((n_un + kRows - 1) / kRows) * kRes; }

// y: [nseries][ypitch] floats holding n_eq = 15 + T rows of 1024 (carried history first); overwritten (it becomes u').
// work: 4 vectors [nseries][wpitch] (v', h, hbar, x), wpitch >= (n_eq + 15) * 1024.  Returns the number of launches.
int launch_lsmr(float *y, long long ypitch, long long T, float *work, long long wpitch, const float *gs, void *scal,
                double *partial, int nseries, int iters, float *series, long long series_pitch, cudaStream_t st)
{
    const long long n_eq = T + kTapsN - 1, n_un = n_eq + kTapsN - 1;
    const int ce = (int)((n_eq + kRows - 1) / kRows), cu = (int)((n_un + kRows - 1) / kRows);
    Scal *sc = static_cast<Scal *>(scal);
    float *v = work, *h = work + (size_t)nseries * wpitch, *hbar = h + (size_t)nseries * wpitch,
          *x = hbar + (size_t)nseries * wpitch;
    const dim3 ge(kRes / kLsmrThreads, ce, nseries), gu(kRes / kLsmrThreads, cu, nseries), gs2(kRes / kLsmrThreads, nseries);
    int n = 0;
    cudaMemsetAsync(sc, 0, lsmr_scalar_bytes(nseries), st);
    u_kernel<-1><<<ge, kLsmrThreads, 0, st>>>(y, ypitch, n_eq, v, wpitch, gs, sc, partial, ce, 1, nullptr, nullptr, nullptr); ++n;
    scalar_kernel<<<gs2, kLsmrThreads, 0, st>>>(sc, partial, ce, 0); ++n;
    v_kernel<<<gu, kLsmrThreads, 0, st>>>(v, wpitch, n_un, y, ypitch, n_eq, gs, sc, partial, cu, 1); ++n;
    scalar_kernel<<<gs2, kLsmrThreads, 0, st>>>(sc, partial, cu, 1); ++n;
    h_kernel<<<gu, kLsmrThreads, 0, st>>>(h, hbar, x, v, wpitch, n_un, sc, 1, 0, nullptr, 0, 0, 0); ++n;
    // The h / hbar / x update of iteration k-1 rides on the u pass of iteration k (rows 0 .. n_eq-1) plus a 15-row launch;
    // x is updated every other iteration (xmode 1 = deferred, 2 = two terms); the last update is a full h_kernel that
    // writes the solution straight into the series.
    const dim3 gtail(kRes / kLsmrThreads, 1, nseries);
    int hm = -1;                                        // x-mode of the update that is still to be done, -1: none
    bool pending = false;                               // an x term of an earlier iteration is still to be applied
    for (int k = 0; k < iters; ++k) {
        if (hm == 1) u_kernel<1><<<ge, kLsmrThreads, 0, st>>>(y, ypitch, n_eq, v, wpitch, gs, sc, partial, ce, 0, h, hbar, x);
        else if (hm == 2) u_kernel<2><<<ge, kLsmrThreads, 0, st>>>(y, ypitch, n_eq, v, wpitch, gs, sc, partial, ce, 0, h, hbar, x);
        else u_kernel<-1><<<ge, kLsmrThreads, 0, st>>>(y, ypitch, n_eq, v, wpitch, gs, sc, partial, ce, 0, nullptr, nullptr, nullptr);
        ++n;
        if (hm >= 0) { h_kernel<<<gtail, kLsmrThreads, 0, st>>>(h, hbar, x, v, wpitch, n_un, sc, 0, hm, nullptr, 0, 0, n_eq); ++n; }
        scalar_kernel<<<gs2, kLsmrThreads, 0, st>>>(sc, partial, ce, 2); ++n;
        v_kernel<<<gu, kLsmrThreads, 0, st>>>(v, wpitch, n_un, y, ypitch, n_eq, gs, sc, partial, cu, 0); ++n;
        scalar_kernel<<<gs2, kLsmrThreads, 0, st>>>(sc, partial, cu, 3); ++n;
        const bool last = (k == iters - 1);
        const int xmode = pending ? 2 : (last ? 0 : 1);
        pending = (xmode == 1);
        if (last) { h_kernel<<<gu, kLsmrThreads, 0, st>>>(h, hbar, x, v, wpitch, n_un, sc, 0, xmode, series, series_pitch, T, 0); ++n; }
        else hm = xmode;                                 // done by the next u pass
    }
    return cudaGetLastError() == cudaSuccess ? n : -1;
}

}  // namespace lofar
