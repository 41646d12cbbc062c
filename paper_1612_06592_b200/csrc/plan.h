// plan.h -- internal plan object and the launcher prototypes of the kernel translation units.
// Not part of the public boundary (include/lofar_moon.h).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <vector>

#include "../../include/lofar_moon.h"

namespace lofar {

// ---- launch parameter blocks -------------------------------------------------------------------
struct BeamformArgs {
    const void *X;        // [S][2][K][xpitch] complex ints
    long long xpitch;     // samples per input row
    long long t0;         // first slice of this launch inside X rows
    long long nt;         // slices to process
    float2 *Z;            // [nz][K][zpitch], slice t0+i stored at column i
    long long zpitch;
    int ztile;            // 1: plan scratch layout [nz][zpitch/16][K][16] (16-slice tiles contiguous over sub-bands)
    const float2 *W;      // [K][B][S] weights (de-dispersion phase folded in when D == 1)
    const float2 *Dph;    // [D][K] trial phasors, used when nphase > 0
    int S, K, B;
    int nphase;           // 0: write the B beam sums; D > 0: write B*D phased series (stage call, D > 1)
    int dtype;            // LOFAR_CI8 / LOFAR_CI16
};

struct IppfArgs {
    const float2 *Z;      // [nz][K][zpitch]
    long long zpitch;
    int ztile;            // 1: [nz][zpitch/16][K][16]: one step of one series is one contiguous K*128-byte block
    long long nc;         // slices in this launch (columns 0..nc-1 of Z)
    float *series;        // [nseries][series_pitch]; this launch writes samples out0 .. out0 + nc*1024
    long long series_pitch;
    long long out0;
    const float2 *Dph;    // [D][K]; applied on load when zmap_trials != 0
    int zmap_trials;      // 0: Z holds one row set per series;  D: Z holds per-beam sums, series = b*D+d
    int K, k0, nseries;
    int nspans, span_len; // span_len is a multiple of 16
    const float *hist_in; // [nseries][15][1024]
    float *hist_out;
    const float2 *gs;     // [16][512] synthesis taps (g[2n + 1024 t], g[2n+1 + 1024 t])
    const float2 *tw;     // twiddles: w1024[256] (pre-pass), TB[32][16] = exp(2 pi i j r / 512) (radix-32 pass)
    double *partial;      // [nseries][partial_pitch] sum of xhat^2 per CTA
    int partial_pitch, partial0;
    float *chunkmax;      // [nseries][chunkmax_pitch] max |xhat| per 16-slice step
    long long chunkmax_pitch, step0;
    int vec_ok;           // Z rows are 16-byte aligned at every step start (128-byte bulk copies allowed)
    // threshold known before the block (causal sigma): candidates are emitted from the FIR epilogue
    const float *thr;     // [nseries] kappa * sigma_ref, or nullptr
    const float *sigma_ref;
    lofar_candidate *cand;
    uint32_t *count;
    uint32_t cap;
    int D;                // trials per beam (candidate.trial = series % D)
    uint64_t offset;      // stream offset of sample 0 of the block
    float *yout;          // nullptr, or [nseries][yout_pitch] float: the inverse-DFT rows y[q][1024] (LSMR inversion, f1);
    long long yout_pitch; //   the FIR is skipped and no series is written
};

// Series-free two-pass trigger (series == NULL, sigma of this block): the flagged (beam, 16-slice step) items are
// recomputed from X -- SIMT beam sums, transform, FIR -- and compared with kappa * sigma.
struct RescanArgs {
    const void *X; long long xpitch; int dtype;      // [S][2][K][xpitch] complex ints, T = slices of the block
    long long T;
    const float2 *W;      // [K][B][S]
    const float2 *Dph;    // [D][K] (applied when D > 1)
    int S, K, k0, B, D;
    const float *hist0;   // [nseries][15][1024] history at the start of the block
    const float2 *gs, *tw;
    const int2 *items;    // (beam, step) list
    const uint32_t *nitems;
    uint32_t items_cap;
    const float *sigma;   // [nseries] of this block
    float kappa;
    const float *chunkmax; long long chunkmax_pitch;
    lofar_candidate *cand; uint32_t *count; uint32_t cap;
    uint64_t offset;
};

struct TriggerArgs {
    const float *series;  // [nseries][series_pitch]
    long long series_pitch;
    long long N;          // samples per series in this block
    int B, D, W;          // beams, trials, envelope window
    float kappa;
    const float *tail;    // [nseries][W-1] samples preceding the block (W > 1)
    double *partial;      // [nseries][partial_pitch]
    int partial_pitch, nparts;
    float *chunkmax;      // [nseries][chunkmax_pitch], one per 16384 samples
    long long chunkmax_pitch, nchunks;
    float *sigma;         // [nseries]
    lofar_candidate *cand;
    uint32_t *count;
    uint32_t cap;
    uint64_t offset;      // stream offset of sample 0 of this block
    const float *sigma_thr;   // [nseries] level the candidates are measured against (= sigma, or the previous block's)
    int zero_count;       // sigma_kernel resets *count (not when candidates were emitted by the inverse PPF)
    int2 *items;          // flagged (beam, 16384-sample chunk) list and its length
    uint32_t *nitems;
    uint32_t items_cap;
};


// Exact de-dispersion (dedisp.cu, f2)
struct DedispArgs {
    const float *xlead;   // [B][xpitch]: two carried slices, then the T slices of this block (undispersed xhat)
    long long xpitch, nlead;   // nlead = T + 2 slices
    float *series;        // [B*D][series_pitch]: output, one slice behind the input
    long long series_pitch, T;
    int B, D;
    const float2 *Dtab;   // [D][8193] exp(-2 pi i 1.343e9 STEC_d / f_j)
    const float2 *tw8192; // [8192] exp(2 pi i m / 8192)
    const float2 *tw16k;  // [4097] exp(2 pi i j / 16384)
    const float2 *tw512;  // TB[32][16] of the 512-point FFT
};

// kernel launchers (each returns the number of kernels it launched, or -1 on a launch error)
int launch_beamform(const BeamformArgs &a, cudaStream_t st);
int launch_ippf(const IppfArgs &a, cudaStream_t st);
int launch_requantize(const float2 *Z, long long n_per_g, int G, float scale, void *X2, cudaStream_t st);
// tensor-core beamformer (beamform_tc.cu)
bool tc_supported(const BeamformArgs &a);
size_t tc_image_halfs(int S, int B);
void tc_build_image(const double *w_re, const double *w_im, int S, int B, unsigned short *hi, unsigned short *lo);
int launch_beamform_tc(const BeamformArgs &a, const void *wimg, cudaStream_t st);
int tc_configure();                                     // opt in to the large dynamic shared memory (current device)
int ippf_configure();                                   // opt in to the large dynamic shared memory
int launch_rescan(const RescanArgs &a, int grid, cudaStream_t st);
int dedisp_configure();
int launch_dedisp(const DedispArgs &a, cudaStream_t st);
// LSMR inversion (lsmr.cu)
size_t lsmr_scalar_bytes(int nseries);
size_t lsmr_partial_count(int nseries, long long n_un);
int launch_lsmr(float *y, long long ypitch, long long T, float *work, long long wpitch, const float *gs, void *scal,
                double *partial, int nseries, int iters, float *series, long long series_pitch, cudaStream_t st);
int launch_trigger_reduce(const TriggerArgs &a, cudaStream_t st);   // sum e^2 + chunk max from the series
int launch_trigger_sigma(const TriggerArgs &a, cudaStream_t st);    // sigma from the partial sums
int launch_trigger_flag(const TriggerArgs &a, cudaStream_t st);     // list of chunks whose maximum can reach the threshold
int launch_trigger_scan(const TriggerArgs &a, int grid, cudaStream_t st);   // threshold scan of the flagged chunks
int launch_trigger_sort(const TriggerArgs &a, bool unique, cudaStream_t st);   // order (and best-trial dedupe)
int launch_sigma_ref(const float *sigma, float kappa, int nseries, float *sigma_ref, float *thr, cudaStream_t st);
int launch_cluster(const lofar_candidate *cand, const uint32_t *count, uint32_t cap, int D, uint64_t gap,
                   lofar_event *events, uint32_t *nevents, uint32_t max_events, cudaStream_t st);
int launch_tail_save(const float *series, long long pitch, long long N, int nseries, int W,
                     float *tail, cudaStream_t st);

}  // namespace lofar

struct lofar_plan {
    int ninv() const { return dedisp == LOFAR_DEDISP_EXACT ? B : B * D; }   // series through the inverse PPF
    // problem
    int S = 0, K = 0, B = 0, D = 1, P = 16, M = 1024, k0 = 0;
    double f_zone = 100e6, clock = 200e6;
    std::vector<double> tau, stec, h;
    lofar_dtype dtype = LOFAR_CI8;
    int max_slices = 0;
    double kappa = 6.0;
    int env_window = 1;
    uint32_t max_cand = 65536;
    int dedisp = LOFAR_DEDISP_SUBBAND;         // f2: LOFAR_DEDISP_EXACT de-disperses the reconstructed 5 ns series per trial
    int inversion = LOFAR_INV_MATCHED;         // f1: LOFAR_INV_LSMR solves H x = y by LSMR instead of applying H^T
    int lsmr_iters = 25;
    int sigma_mode = LOFAR_SIGMA_BLOCK;        // f3: LOFAR_SIGMA_CAUSAL judges block i against sigma of block i-1
    std::vector<float> sigma_init, thr_init;   // optional reference level of the first block of a stream (and kappa times it)
    // device memory: every plan-owned device buffer goes through these (lofar_plan_set_allocator)
    void *(*alloc_fn)(size_t, void *) = nullptr;
    void (*free_fn)(void *, void *) = nullptr;
    void *alloc_ctx = nullptr;
    size_t scratch_limit = (size_t)16 << 30;  // bytes of beam-sum scratch (all slots together); sized for 180 GB of HBM
    // Two-lane block pipeline (lofar_plan_set_overlap): the beamformer of chunk c+1 runs on a low-priority stream
    // beside the inverse PPF of chunk c, on the SMs the inverse PPF leaves free; two scratch slots.
    int overlap = 0;                   // requested: 0 = serial (default: measured faster), 1 = pipeline
    long long overlap_chunk = 8192;    // slices per chunk of the pipeline (fill + drain = one chunk of each kernel)
    bool lanes_active = false;         // the block call in progress uses the pipeline (more than one chunk)
    bool overlap_on = false;           // decided by build(): tensor-core beamformer and at least two chunks
    int ippf_sms = 148;                // SMs the inverse-PPF spans are planned for (num_sms minus the reserve)
    cudaStream_t s_bf = nullptr, s_ippf = nullptr;
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr, ev_bf[2] = {nullptr, nullptr}, ev_ippf[2] = {nullptr, nullptr};
    // device state
    bool built = false;
    bool reset_pending = false;        // carried state is zeroed on the stream of the next compute call
    int num_sms = 148;
    unsigned short *dWimg = nullptr;   // [K][2][image] fp16 hi/lo operand images for the tensor-core beamformer
    int tc_min_beams = 4;              // use tcgen05 from this many beams on (int8 input)
    float2 *dW = nullptr, *dDph = nullptr, *dGs = nullptr, *dTw = nullptr;
    float *dHist[2] = {nullptr, nullptr};
    int hist_parity = 0;
    float *dTail = nullptr;
    float2 *dZ = nullptr;
    long long zchunk = 0;          // slices per scratch chunk
    double *dPartial = nullptr;
    int partial_pitch = 0;
    float *dChunkMax = nullptr;
    long long chunkmax_pitch = 0;
    int2 *dItems = nullptr;            // flagged (beam, chunk) list of the trigger
    uint32_t *dNItems = nullptr;
    uint32_t items_cap = 0;
    float *dSigmaRef = nullptr, *dThr = nullptr;   // causal sigma: level of the previous block and kappa times it
    bool have_ref = false;
    float *dHist0 = nullptr;           // history at the start of the block (series-free two-pass trigger)
    float *dY = nullptr, *dLsmrWork = nullptr;     // LSMR: inverse-DFT rows [ns][15+T][1024]; v', h, hbar, x [4][ns][T+30][1024]
    long long ypitch = 0, wpitch = 0;
    void *dLsmrScal = nullptr;
    float *dXhat = nullptr;            // exact de-dispersion: [B][2 + T][1024] undispersed series behind two carried slices
    long long xhat_pitch = 0;
    float2 *dDtab = nullptr, *dTw8192 = nullptr, *dTw16k = nullptr;
    double *dLsmrPartial = nullptr;
    size_t device_bytes = 0;
    uint64_t offset = 0;
    uint64_t launches = 0;
    // streaming
    cudaStream_t s_copy = nullptr, s_comp = nullptr;
    void *dX[2] = {nullptr, nullptr};
    size_t dX_bytes = 0;
    cudaEvent_t ev_copied[2] = {nullptr, nullptr}, ev_done[2] = {nullptr, nullptr};
    bool slot_used[2] = {false, false};
    lofar_candidate *dCand[2] = {nullptr, nullptr};
    uint32_t *dCount[2] = {nullptr, nullptr};
    float *dSigma[2] = {nullptr, nullptr};
    uint32_t *hCount = nullptr;    // pinned, one per push since the last sync (ring of 64)
    int pushes = 0;
    uint64_t push_index = 0;
    // per-kernel profiling (lofar_plan_profile)
    bool prof = false;
    struct ProfRec { int id; cudaEvent_t a, b; };
    std::vector<ProfRec> prof_pending;
    std::vector<cudaEvent_t> prof_pool;
};
