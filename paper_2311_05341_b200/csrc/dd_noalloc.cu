// dd_noalloc.cu -- dd_execute_noalloc: the transform for callers that must not allocate device memory.
//
// Who this is for.  Every other way into the library goes through dd_plan_create, which cudaMallocs the
// plan's tiling metadata and its lane-interleaved workspace.  Two kinds of caller cannot do that:
//   * a process that has already handed the whole device to its own pool (a telescope back end that
//     reserves the GPU at start-up, a framework's caching allocator grown to the card's capacity):
//     cudaMalloc simply fails there with out-of-memory;
//   * a real-time stage between two blocks of an observation: cudaMalloc and cudaFree synchronise the
//     whole device, so one call stalls every other stream of the pipeline for an unbounded time.
// For them this file holds a direct form of the dedispersion kernel (Eq. 3; Alg. 1,
// 72-76) whose only scratch -- the device copy of the integer shift table s(d,c) -- lives in a
// file-scope __device__ array that is part of the loaded library image.  It is a small-problem path
// (one global-memory read per add, no shared-memory tiling): use a plan whenever you may allocate.
//
// Shares no state with the plan-based path and changes none of it.
#include <cuda_runtime.h>

#include <cstdint>
#include <mutex>

#include "dd.h"

namespace {

// The scratch.  DD_NOALLOC_MAX_TABLE int32 entries (4 MiB): every GPU on which this library's image is
// loaded carries it from then until the process exits, used or not.  In HOST code the name `g_table` is
// only a handle for the runtime's symbol calls -- it is not a device address, and a kernel handed
// `g_table` from the host would fault or (where the GPU can reach host memory) scribble somewhere else.
// Host code must ask for the address: device_table() below.
static __device__ __align__(256) int32_t g_table[DD_NOALLOC_MAX_TABLE];

constexpr int kMaxDevices = 64;
std::mutex g_setup_mutex;
int32_t *g_table_addr[kMaxDevices] = {};  // device address of g_table on device i (null: not asked yet)
int g_device_ok[kMaxDevices] = {};        // 1 after the compute-capability check passed

// Per-device set-up: with `device` current, resolve the device address of g_table once and keep it.
// No allocation: cudaGetSymbolAddress looks the array up in the module the runtime has loaded.
int device_table(int device, int32_t **ptr)
{
    if (device < 0 || device >= kMaxDevices) return DD_ERR_UNSUPPORTED_DEVICE;
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    if (!g_device_ok[device]) {
        int major = 0;
        if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, device) != cudaSuccess) {
            cudaGetLastError();
            return DD_ERR_CUDA;
        }
        if (major != 10) return DD_ERR_UNSUPPORTED_DEVICE;
        g_device_ok[device] = 1;
    }
    if (!g_table_addr[device]) {
        void *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_table);
        if (e != cudaSuccess || !p) {
            cudaGetLastError();
            return DD_ERR_CUDA;
        }
        g_table_addr[device] = static_cast<int32_t *>(p);
    }
    *ptr = g_table_addr[device];
    return DD_OK;
}

constexpr int kThreads = 256;
constexpr int kPerThread = 4;  // output samples per thread, kThreads apart (coalesced rows)

template <int MODE> struct SampleOf;
template <> struct SampleOf<DD_U8> {
    using acc_t = uint32_t;
    static __device__ __forceinline__ acc_t load(const void *in, int64_t row, int64_t t)
    { return __ldg(static_cast<const uint8_t *>(in) + row + t); }
    static __device__ __forceinline__ int64_t row_elems(int64_t nsamps) { return nsamps; }
};
template <> struct SampleOf<DD_U16> {
    using acc_t = uint32_t;
    static __device__ __forceinline__ acc_t load(const void *in, int64_t row, int64_t t)
    { return __ldg(static_cast<const uint16_t *>(in) + row + t); }
    static __device__ __forceinline__ int64_t row_elems(int64_t nsamps) { return nsamps; }
};
template <> struct SampleOf<DD_F32> {
    using acc_t = float;
    static __device__ __forceinline__ acc_t load(const void *in, int64_t row, int64_t t)
    { return __ldg(static_cast<const float *>(in) + row + t); }
    static __device__ __forceinline__ int64_t row_elems(int64_t nsamps) { return nsamps; }
};
template <> struct SampleOf<DD_U4> {  // two samples per byte, the earlier one in the low nibble (dd.h)
    using acc_t = uint32_t;
    static __device__ __forceinline__ acc_t load(const void *in, int64_t row, int64_t t)
    {
        const uint32_t b = __ldg(static_cast<const uint8_t *>(in) + row + (t >> 1));
        return (b >> (4u * static_cast<uint32_t>(t & 1))) & 15u;
    }
    static __device__ __forceinline__ int64_t row_elems(int64_t nsamps) { return nsamps >> 1; }
};

// out[d][t] = sum_c in[c][t + s(d,c)], one DM trial and kThreads*kPerThread output samples per thread
// block, channels in ascending order.  `table` is the address device_table() returned.
template <int MODE>
__global__ void __launch_bounds__(kThreads)
dedisperse_direct_kernel(const int32_t *__restrict__ table, const void *__restrict__ in,
                         typename SampleOf<MODE>::acc_t *__restrict__ out, int nchans, int64_t nsamps,
                         int64_t out_len, int64_t tiles_per_dm)
{
    using S = SampleOf<MODE>;
    const int64_t blk = static_cast<int64_t>(blockIdx.x);
    const int64_t d = blk / tiles_per_dm;
    const int64_t t0 = (blk - d * tiles_per_dm) * (kThreads * kPerThread) + threadIdx.x;
    const int32_t *__restrict__ row_shift = table + d * nchans;
    const int64_t pitch = S::row_elems(nsamps);

    typename S::acc_t acc[kPerThread];
#pragma unroll
    for (int k = 0; k < kPerThread; ++k) acc[k] = 0;
    for (int c = 0; c < nchans; ++c) {
        const int64_t s = __ldg(row_shift + c);  // the same word for the whole block
        const int64_t row = static_cast<int64_t>(c) * pitch;
#pragma unroll
        for (int k = 0; k < kPerThread; ++k) {
            const int64_t t = t0 + k * kThreads;
            if (t < out_len) acc[k] += S::load(in, row, t + s);
        }
    }
#pragma unroll
    for (int k = 0; k < kPerThread; ++k) {
        const int64_t t = t0 + k * kThreads;
        if (t < out_len) out[d * out_len + t] = acc[k];
    }
}

template <int MODE>
cudaError_t launch(const int32_t *table, const void *d_in, void *d_out, int ndm, int nchans, int64_t nsamps,
                   int64_t out_len, cudaStream_t st)
{
    const int64_t tiles = (out_len + kThreads * kPerThread - 1) / (kThreads * kPerThread);
    const int64_t blocks = tiles * ndm;
    if (blocks > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    dedisperse_direct_kernel<MODE><<<static_cast<unsigned>(blocks), kThreads, 0, st>>>(
        table, d_in, static_cast<typename SampleOf<MODE>::acc_t *>(d_out), nchans, nsamps, out_len, tiles);
    return cudaGetLastError();
}

}  // namespace

extern "C" int dd_execute_noalloc(const int32_t *table, int ndm, int nchans, int64_t nsamps, int in_dtype,
                                  const void *d_in, void *d_out, void *cuda_stream)
{
    if (!table || !d_in || !d_out || ndm <= 0 || nchans <= 0 || nsamps <= 0) return DD_ERR_INVALID_ARG;
    if (in_dtype != DD_U8 && in_dtype != DD_U16 && in_dtype != DD_F32 && in_dtype != DD_U4)
        return DD_ERR_INVALID_ARG;
    if (in_dtype == DD_U4 && (nsamps & 1)) return DD_ERR_INVALID_ARG;
    const int64_t entries = static_cast<int64_t>(ndm) * nchans;
    if (entries > DD_NOALLOC_MAX_TABLE) return DD_ERR_STATIC_LIMIT;
    if (in_dtype == DD_U16 && 65535LL * nchans >= (1LL << 32)) return DD_ERR_OVERFLOW;

    int32_t max_shift = 0;
    for (int64_t i = 0; i < entries; ++i) {
        if (table[i] < 0) return DD_ERR_INVALID_ARG;
        if (table[i] > max_shift) max_shift = table[i];
    }
    if (max_shift >= nsamps) return DD_ERR_SHIFT_TOO_LARGE;
    const int64_t out_len = nsamps - max_shift;

    int device = -1;
    if (cudaGetDevice(&device) != cudaSuccess) {
        cudaGetLastError();
        return DD_ERR_CUDA;
    }
    int32_t *d_table = nullptr;
    const int rc = device_table(device, &d_table);
    if (rc != DD_OK) return rc;

    // Every entry the kernel reads is overwritten here, so nothing in the array has to start at zero and
    // whatever an earlier call left beyond `entries` is never looked at.  A pageable source is staged by
    // the runtime before this returns, so `table` is the caller's again on return.
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    if (cudaMemcpyAsync(d_table, table, static_cast<size_t>(entries) * sizeof(int32_t), cudaMemcpyHostToDevice,
                        st) != cudaSuccess) {
        cudaGetLastError();
        return DD_ERR_CUDA;
    }
    cudaError_t e = cudaSuccess;
    switch (in_dtype) {
    case DD_U8: e = launch<DD_U8>(d_table, d_in, d_out, ndm, nchans, nsamps, out_len, st); break;
    case DD_U16: e = launch<DD_U16>(d_table, d_in, d_out, ndm, nchans, nsamps, out_len, st); break;
    case DD_F32: e = launch<DD_F32>(d_table, d_in, d_out, ndm, nchans, nsamps, out_len, st); break;
    default: e = launch<DD_U4>(d_table, d_in, d_out, ndm, nchans, nsamps, out_len, st); break;
    }
    return e == cudaSuccess ? DD_OK : DD_ERR_CUDA;
}
