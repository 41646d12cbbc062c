// noalloc.cu -- lofar_trigger_static: the stand-alone threshold trigger (step a5; definitions
// O7 / O8 in DESIGN.md) for callers that may not allocate: code under CUDA graph capture, tight serving loops,
// harnesses that forbid cudaMalloc.  Same kernels and the same arithmetic as lofar_trigger (trigger.cu: reduce ->
// sigma -> flag -> scan -> sort), but no plan and no allocation of any kind: the scratch the kernels need (per-chunk
// sums of squares and maxima, the list of flagged chunks and its counter) lives in ONE file-scope device array of
// fixed size.  Every GPU that loads the library holds that array (about 6.1 MiB) until the process exits.
//
// The array's name is a host-side stand-in in host code, not a device address: its address is taken once per device
// with cudaGetSymbolAddress (that device current, return code checked) and passed to the kernels.
//
// All calls share the array and it keeps the last call's contents.  What must start at zero -- the candidate
// counter and the flag-list counter -- is cleared on the stream by sigma_kernel at the start of every call; the
// per-chunk entries are overwritten for exactly the range a call uses.  Two calls that overlap on the GPU (different
// streams without an ordering between them) race on the array: callers serialise them.
#include <mutex>

#include "plan.h"

namespace lofar {
namespace {

constexpr long long kStaticChunk = 16384;                       // samples per pruning chunk (trigger.cu: kChunk)
constexpr long long kStaticMaxChunks = LOFAR_STATIC_MAX_CHUNKS; // over all series of one call
constexpr uint32_t kStaticItems = 16384;                        // flagged chunks before the scan falls back to all
constexpr int kMaxDevices = 64;

// section offsets, each 256-byte aligned
constexpr size_t kOffPartial = 0;                                                    // double[kStaticMaxChunks]
constexpr size_t kOffChunkMax = kOffPartial + (size_t)kStaticMaxChunks * sizeof(double);   // float[kStaticMaxChunks]
constexpr size_t kOffItems = kOffChunkMax + (size_t)kStaticMaxChunks * sizeof(float);      // int2[kStaticItems]
constexpr size_t kOffNItems = kOffItems + (size_t)kStaticItems * sizeof(int2);             // uint32_t (+ padding)
constexpr size_t kStaticBytes = kOffNItems + 256;
static_assert(kOffChunkMax % 256 == 0 && kOffItems % 256 == 0 && kOffNItems % 256 == 0, "sections stay 256-byte aligned");

static __device__ __align__(256) unsigned char g_static_scratch[kStaticBytes];

std::mutex g_mutex;
unsigned char *g_addr[kMaxDevices];      // device address of g_static_scratch on each device, nullptr = not yet asked

// Once per device, with that device current: the device address of the array.
lofar_status scratch_address(unsigned char **out)
{
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return LOFAR_E_CUDA;
    if (dev < 0 || dev >= kMaxDevices) return LOFAR_E_STATE;
    std::lock_guard<std::mutex> lock(g_mutex);
    if (!g_addr[dev]) {
        void *p = nullptr;
        if (cudaGetSymbolAddress(&p, g_static_scratch) != cudaSuccess || !p) return LOFAR_E_CUDA;
        g_addr[dev] = static_cast<unsigned char *>(p);
    }
    *out = g_addr[dev];
    return LOFAR_OK;
}

}  // namespace
}  // namespace lofar

using namespace lofar;

extern "C" {

lofar_status lofar_trigger_static(const float *series, int nseries, int64_t samples, int64_t series_pitch, double kappa,
                                  uint64_t offset, lofar_candidate *cand, uint32_t max_candidates, uint32_t *count,
                                  float *sigma, void *stream)
{
    if (!series || !cand || !count || !sigma) return LOFAR_E_INVALID;
    if (nseries <= 0 || samples <= 0 || series_pitch < samples || !(kappa > 0.0) || max_candidates == 0) return LOFAR_E_INVALID;
    const long long nchunks = (samples + kStaticChunk - 1) / kStaticChunk;
    // beyond the fixed scratch: LOFAR_E_SHAPE, nothing is launched (lofar_status_string: "shape out of range")
    if (nchunks > kStaticMaxChunks || (long long)nseries * nchunks > kStaticMaxChunks) return LOFAR_E_SHAPE;
    unsigned char *base = nullptr;
    const lofar_status s = scratch_address(&base);
    if (s != LOFAR_OK) return s;
    cudaStream_t st = static_cast<cudaStream_t>(stream);

    TriggerArgs t{};
    t.series = series; t.series_pitch = series_pitch; t.N = samples;
    t.B = nseries; t.D = 1; t.W = 1; t.kappa = (float)kappa;
    t.tail = nullptr;
    t.partial = reinterpret_cast<double *>(base + kOffPartial); t.partial_pitch = (int)nchunks; t.nparts = (int)nchunks;
    t.chunkmax = reinterpret_cast<float *>(base + kOffChunkMax); t.chunkmax_pitch = nchunks; t.nchunks = nchunks;
    t.sigma = sigma; t.cand = cand; t.count = count; t.cap = max_candidates;
    t.offset = offset;
    t.sigma_thr = sigma;
    t.zero_count = 1;                                // sigma_kernel clears *count and the flag-list counter
    t.items = reinterpret_cast<int2 *>(base + kOffItems);
    t.nitems = reinterpret_cast<uint32_t *>(base + kOffNItems);
    t.items_cap = kStaticItems;

    int sms = 148, dev = 0;
    if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (launch_trigger_reduce(t, st) < 0) return LOFAR_E_CUDA;
    if (launch_trigger_sigma(t, st) < 0) return LOFAR_E_CUDA;
    if (launch_trigger_flag(t, st) < 0) return LOFAR_E_CUDA;
    if (launch_trigger_scan(t, 4 * sms, st) < 0) return LOFAR_E_CUDA;
    if (launch_trigger_sort(t, false, st) < 0) return LOFAR_E_CUDA;
    return LOFAR_OK;
}

}  // extern "C"
