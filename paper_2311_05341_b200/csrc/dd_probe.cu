// dd_probe.cu -- measured on-chip peaks of the device the library runs on (dd_probe in dd.h).
//
// The dedispersion kernels are bound by the shared-memory pipe and, next, by the integer ALUs
// (DESIGN.md "Rooflines"); the paper computes both peaks from data-sheet numbers (Eq. 8 and
// Eq. 9).  MEASURED_PEAKS.json has neither, so the library measures them:
//   * shared-memory read bandwidth with LDS.32 / LDS.64 / LDS.128, conflict-free, no consumer;
//   * lane-instruction rates of the instructions the kernels accumulate with;
//   * tensor-memory read bandwidth alone and next to shared-memory reads (the question behind
//     DESIGN.md's "TMEM as a second operand store");
//   * the SM clock while doing so.
// Every probe runs one CTA per SM (148 x 1024 threads, 8 warps per scheduler), times its
// loop with clock64() inside the kernel and reports the median over CTAs, per clock per SM.
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdint>
#include <vector>

#include "dd.h"

namespace {

constexpr int kThreads = 1024;
constexpr int kIter = 2048;
constexpr int kChains = 8;

// ---------------------------------------------------------------- lane-instruction rates
template <int OP>
__device__ __forceinline__ void lane_op(uint32_t &a, uint32_t x, uint32_t y)
{
    // IADD3: y = another chain's accumulator, a true three-input add; IMAD_HI: x = another chain's
    // accumulator (ptxas hoists the high half of a loop-invariant product)
    if (OP == DD_PROBE_IADD3)
        asm volatile("{ .reg .u32 t; add.u32 t, %1, %2; add.u32 %0, %0, t; }" : "+r"(a) : "r"(x), "r"(y));
    else if (OP == DD_PROBE_VIADD16X2)
        a = __vadd2(a, x);
    else if (OP == DD_PROBE_IMAD)
        asm volatile("mad.lo.u32 %0, %1, %2, %0;" : "+r"(a) : "r"(x), "r"(y));
    else if (OP == DD_PROBE_FADD)
        asm volatile("{ .reg .f32 f, g; mov.b32 f, %0; mov.b32 g, %1; add.rn.f32 f, f, g; mov.b32 %0, f; }"
                     : "+r"(a)
                     : "r"(x));
    else if (OP == DD_PROBE_LOP3)
        asm volatile("lop3.b32 %0, %0, %1, %2, 0xEA;" : "+r"(a) : "r"(x), "r"(y));
    else if (OP == DD_PROBE_PRMT)
        asm volatile("prmt.b32 %0, %0, %1, 0x4341;" : "+r"(a) : "r"(x));
    else if (OP == DD_PROBE_SHIFT_ADD)
        asm volatile("{ .reg .u32 t; shr.u32 t, %1, 4; add.u32 %0, %0, t; }" : "+r"(a) : "r"(x));
    else if (OP == DD_PROBE_IMAD_HI)
        asm volatile("mad.hi.u32 %0, %1, %2, %0;" : "+r"(a) : "r"(x), "r"(y));
    else if (OP == DD_PROBE_IDP4A)
        asm volatile("dp4a.u32.u32 %0, %1, %2, %0;" : "+r"(a) : "r"(x), "r"(y));
    else if (OP == DD_PROBE_SHF)
        asm volatile("shf.r.wrap.b32 %0, %0, %1, 8;" : "+r"(a) : "r"(x));
}

template <int OP>
__global__ void __launch_bounds__(kThreads, 1) lane_rate_kernel(uint32_t *sink, long long *cycles, uint32_t seed)
{
    uint32_t a[kChains];
    // operands the compiler knows nothing about (the host fills `sink` before the launch)
    const uint32_t x = sink[threadIdx.x] ^ seed, y = sink[kThreads + threadIdx.x] | 1u;
#pragma unroll
    for (int i = 0; i < kChains; ++i) a[i] = sink[2 * kThreads + threadIdx.x] + i;
    __syncthreads();
    const long long t0 = clock64();
#pragma unroll 1
    for (int it = 0; it < kIter; ++it) {
#pragma unroll
        for (int u = 0; u < 4; ++u)
#pragma unroll
            for (int i = 0; i < kChains; ++i)
                lane_op<OP>(a[i], OP == DD_PROBE_IMAD_HI ? a[(i + 1) % kChains] : x,
                            OP == DD_PROBE_IADD3 ? a[(i + 1) % kChains] : y);
    }
    __syncthreads();
    const long long t1 = clock64();
    uint32_t s = 0;
#pragma unroll
    for (int i = 0; i < kChains; ++i) s += a[i];
    sink[blockIdx.x * kThreads + threadIdx.x] = s;
    if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
}

// ---------------------------------------------------------------- shared-memory read bandwidth
template <int VW>
__global__ void __launch_bounds__(kThreads, 1) lds_kernel(uint32_t *sink, long long *cycles)
{
    extern __shared__ uint32_t sm[];
    for (int i = threadIdx.x; i < 8192; i += kThreads) sm[i] = i;
    __syncthreads();
    // a warp reads 32 consecutive VW-word pieces: every bank once per 128 bytes, no conflicts
    const uint32_t addr = static_cast<uint32_t>(__cvta_generic_to_shared(sm)) + (threadIdx.x & 31) * 4 * VW;
    uint32_t acc = 0;
    const long long t0 = clock64();
#pragma unroll 1
    for (int it = 0; it < kIter; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            uint32_t x0, x1 = 0, x2 = 0, x3 = 0;
            const uint32_t ad = addr + u * 128 * VW;
            if (VW == 1)
                asm volatile("ld.volatile.shared.u32 %0, [%1];" : "=r"(x0) : "r"(ad));
            else if (VW == 2)
                asm volatile("ld.volatile.shared.v2.u32 {%0,%1}, [%2];" : "=r"(x0), "=r"(x1) : "r"(ad));
            else
                asm volatile("ld.volatile.shared.v4.u32 {%0,%1,%2,%3}, [%4];"
                             : "=r"(x0), "=r"(x1), "=r"(x2), "=r"(x3)
                             : "r"(ad));
            if (it == kIter - 1) acc += x0 + x1 + x2 + x3;
        }
    }
    __syncthreads();
    const long long t1 = clock64();
    sink[blockIdx.x * kThreads + threadIdx.x] = acc;
    if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
}

#ifdef DD_TUNING  // experiments of DESIGN.md section 10 (numbers: profiles/r02_peaks.md): libdd_tuning.so only
// ---------------------------------------------------------------- tensor memory next to shared memory
// MODE 0: tcgen05.ld.32x32b.x8 only; 1: the same interleaved with four LDS.64 per iteration (equal bytes)
template <int MODE>
__global__ void __launch_bounds__(512, 1) tmem_kernel(uint32_t *sink, long long *cycles)
{
    extern __shared__ uint32_t sm[];
    __shared__ uint32_t tmem_base;
    for (int i = threadIdx.x; i < 8192; i += blockDim.x) sm[i] = i;
    if (threadIdx.x < 32) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 256;" ::"r"(
            static_cast<uint32_t>(__cvta_generic_to_shared(&tmem_base))));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;");
    const uint32_t tb = tmem_base;
    const int warp = threadIdx.x >> 5;
    const uint32_t taddr = tb + (static_cast<uint32_t>(32 * (warp & 3)) << 16);  // lane quarter of this warp
    for (int c = 0; c < 256; c += 8) {
        const uint32_t z = threadIdx.x + c;
        asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%1,%1,%1,%1,%1,%1,%1};" ::"r"(taddr + c), "r"(z));
    }
    asm volatile("tcgen05.wait::st.sync.aligned;");
    __syncthreads();
    uint32_t a[8] = {0, 1, 2, 3, 4, 5, 6, 7};
    const uint32_t addr = static_cast<uint32_t>(__cvta_generic_to_shared(sm)) + (threadIdx.x & 31) * 8;
    const long long t0 = clock64();
#pragma unroll 1
    for (int it = 0; it < kIter; ++it) {
        const uint32_t col = (it * 8) & 255;
        uint32_t y[8];
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                     : "=r"(y[0]), "=r"(y[1]), "=r"(y[2]), "=r"(y[3]), "=r"(y[4]), "=r"(y[5]), "=r"(y[6]), "=r"(y[7])
                     : "r"(taddr + col));
        if (MODE == 1) {
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                uint32_t x0, x1;
                asm volatile("ld.volatile.shared.v2.u32 {%0,%1}, [%2];" : "=r"(x0), "=r"(x1) : "r"(addr + u * 256));
                a[u] += x0;
                a[u + 4] += x1;
            }
        }
        asm volatile("tcgen05.wait::ld.sync.aligned;");
#pragma unroll
        for (int u = 0; u < 8; ++u) a[u] += y[u];
    }
    __syncthreads();
    const long long t1 = clock64();
    uint32_t s = 0;
    for (int i = 0; i < 8; ++i) s += a[i];
    sink[blockIdx.x * blockDim.x + threadIdx.x] = s;
    if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    if (threadIdx.x < 32) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 256;" ::"r"(tb));
}

// ---------------------------------------------------------------- f32 accumulate fed from two operand stores
// The inner loop a tensor-memory "second operand store" kernel would run,
// without its global-memory side: 16 warps, a thread owns T = 33 consecutive outputs of RD = 2 DM
// trials (lane stride 33 words: conflict-free LDS.32 for any shift).  Per group of 8 channels,
// NT of them are served from tensor memory: the four warps of a lane quarter first copy NT windows
// of WCOL = 128 columns (T + shift span of 8 DMs, rounded up) from shared memory into their quarter
// (LDS.32 + tcgen05.st), meet at a named barrier, then every warp reads its 33 columns per (channel,
// DM) at a warp-uniform offset (tcgen05.ld x32 + x1); the other 8 - NT channels are read from shared
// memory, one LDS.32 per add.  Reports adds per clock per SM.  NT = 0 is the present kernel's loop;
// FILL = false fills the windows once only (the cost of the tensor-memory reads alone).
template <int NT, bool FILL>
__global__ void __launch_bounds__(512, 1) hybrid_kernel(uint32_t *sink, long long *cycles)
{
    constexpr int T = 33, RD = 2, G = 8, WCOL = 128;
    extern __shared__ uint32_t sm[];
    __shared__ uint32_t tmem_base;
    for (int i = threadIdx.x; i < 16384; i += blockDim.x) sm[i] = __float_as_uint(1.0f + (i & 7));
    if (threadIdx.x < 32) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(
            static_cast<uint32_t>(__cvta_generic_to_shared(&tmem_base))));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;");
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, quarter = warp & 3, member = warp >> 2;
    const uint32_t taddr = tmem_base + (static_cast<uint32_t>(32 * quarter) << 16);
    const uint32_t seg = static_cast<uint32_t>(__cvta_generic_to_shared(sm)) + (quarter * 32 + lane) * T * 4;
    float acc[RD][T];
#pragma unroll
    for (int r = 0; r < RD; ++r)
#pragma unroll
        for (int i = 0; i < T; ++i) acc[r][i] = 0.f;
    uint32_t off = sink[threadIdx.x & 31] & 63u;  // warp-uniform pseudo shifts, unknown to the compiler
    off = __shfl_sync(0xffffffffu, off, 0);
    __syncthreads();
    const long long t0 = clock64();
#pragma unroll 1
    for (int it = 0; it < 256; ++it) {
        if (NT > 0) {
            // fill: this warp copies window `member` (and member + 4 when NT = 8) of its quarter
#pragma unroll 1
            for (int wn = member; wn < NT && (FILL || it == 0); wn += 4) {
#pragma unroll 2
                for (int c0 = 0; c0 < WCOL; c0 += 16) {
                    uint32_t v[16];
#pragma unroll
                    for (int i = 0; i < 16; ++i)
                        asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v[i]) : "r"(seg + ((wn * 5 + c0 + i + off) & 1023) * 4));
                    asm volatile(
                        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};" ::"r"(
                            taddr + wn * WCOL + c0),
                        "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]), "r"(v[8]),
                        "r"(v[9]), "r"(v[10]), "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15]));
                }
            }
            asm volatile("tcgen05.wait::st.sync.aligned;");
            asm volatile("tcgen05.fence::before_thread_sync;");
            asm volatile("bar.sync %0, 128;" ::"r"(1 + quarter));
            asm volatile("tcgen05.fence::after_thread_sync;");
#pragma unroll 1
            for (int wn = 0; wn < NT; ++wn)
#pragma unroll
                for (int r = 0; r < RD; ++r) {
                    const uint32_t col = taddr + wn * WCOL + ((off + 7 * r + wn) & 63u);
                    // 33 columns as 16 + 16 + 1 (a 32-column load would need 33 more live registers)
                    uint32_t y[2][16], y32;
#pragma unroll
                    for (int h = 0; h < 2; ++h)
                        asm volatile(
                            "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                            : "=r"(y[h][0]), "=r"(y[h][1]), "=r"(y[h][2]), "=r"(y[h][3]), "=r"(y[h][4]), "=r"(y[h][5]),
                              "=r"(y[h][6]), "=r"(y[h][7]), "=r"(y[h][8]), "=r"(y[h][9]), "=r"(y[h][10]), "=r"(y[h][11]),
                              "=r"(y[h][12]), "=r"(y[h][13]), "=r"(y[h][14]), "=r"(y[h][15])
                            : "r"(col + 16 * h));
                    asm volatile("tcgen05.ld.sync.aligned.32x32b.x1.b32 {%0}, [%1];" : "=r"(y32) : "r"(col + 32));
                    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
                    for (int i = 0; i < 32; ++i) acc[r][i] += __uint_as_float(y[i >> 4][i & 15]);
                    acc[r][32] += __uint_as_float(y32);
                }
            // the windows may be overwritten only after every warp of the quarter has read them
            asm volatile("tcgen05.fence::before_thread_sync;");
            asm volatile("bar.sync %0, 128;" ::"r"(5 + quarter));
        }
#pragma unroll
        for (int ch = NT; ch < G; ++ch)
#pragma unroll
            for (int r = 0; r < RD; ++r) {
                const uint32_t a = seg + ((ch * 11 + r * 3 + off) & 63u) * 4;
#pragma unroll
                for (int i = 0; i < T; ++i) {
                    uint32_t x;
                    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(x) : "r"(a + i * 4));
                    acc[r][i] += __uint_as_float(x);
                }
            }
    }
    __syncthreads();
    const long long t1 = clock64();
    float s = 0.f;
#pragma unroll
    for (int r = 0; r < RD; ++r)
#pragma unroll
        for (int i = 0; i < T; ++i) s += acc[r][i];
    sink[blockIdx.x * blockDim.x + threadIdx.x] = __float_as_uint(s);
    if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    if (threadIdx.x < 32) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem_base));
}
#endif  // DD_TUNING

struct Scratch {
    uint32_t *sink = nullptr;
    long long *cycles = nullptr;
    int nsm = 0;
    ~Scratch()
    {
        cudaFree(sink);
        cudaFree(cycles);
    }
};

// median over CTAs of the in-kernel cycle counts of the second of two launches
template <typename Launch>
int median_cycles(Scratch &s, Launch launch, double *cycles)
{
    for (int r = 0; r < 2; ++r) launch();
    if (cudaDeviceSynchronize() != cudaSuccess) {
        cudaGetLastError();
        return DD_ERR_CUDA;
    }
    std::vector<long long> h(static_cast<size_t>(s.nsm));
    if (cudaMemcpy(h.data(), s.cycles, h.size() * sizeof(long long), cudaMemcpyDeviceToHost) != cudaSuccess)
        return DD_ERR_CUDA;
    std::nth_element(h.begin(), h.begin() + h.size() / 2, h.end());
    *cycles = static_cast<double>(h[h.size() / 2]);
    return DD_OK;
}

template <int OP>
int lane_rate(Scratch &s, double *out)
{
    double cyc = 0;
    const int rc = median_cycles(s, [&] { lane_rate_kernel<OP><<<s.nsm, kThreads>>>(s.sink, s.cycles, 12345u); }, &cyc);
    if (rc == DD_OK) *out = static_cast<double>(kThreads) * kIter * 4 * kChains / cyc;
    return rc;
}

template <int VW>
int lds_rate(Scratch &s, double *out)
{
    double cyc = 0;
    const int rc = median_cycles(s, [&] { lds_kernel<VW><<<s.nsm, kThreads, 32768>>>(s.sink, s.cycles); }, &cyc);
    if (rc == DD_OK) *out = static_cast<double>(kThreads) * kIter * 8 * (4 * VW) / cyc;
    return rc;
}

#ifdef DD_TUNING
template <int MODE>
int tmem_rate(Scratch &s, double *out)
{
    double cyc = 0;
    const int rc = median_cycles(s, [&] { tmem_kernel<MODE><<<s.nsm, 512, 32768>>>(s.sink, s.cycles); }, &cyc);
    // per iteration a thread reads 8 words from TMEM (and, MODE 1, 8 words from shared memory)
    if (rc == DD_OK) *out = 512.0 * kIter * 32 / cyc;
    return rc;
}

template <int NT, bool FILL>
int hybrid_rate(Scratch &s, double *out)
{
    double cyc = 0;
    if (cudaFuncSetAttribute(reinterpret_cast<const void *>(hybrid_kernel<NT, FILL>), cudaFuncAttributeMaxDynamicSharedMemorySize,
                             65536 + 8192) != cudaSuccess)
        return DD_ERR_CUDA;
    if (cudaMemset(s.cycles, 0, static_cast<size_t>(s.nsm) * sizeof(long long)) != cudaSuccess) return DD_ERR_CUDA;
    const int rc = median_cycles(s, [&] { hybrid_kernel<NT, FILL><<<s.nsm, 512, 65536 + 8192>>>(s.sink, s.cycles); }, &cyc);
    if (rc == DD_OK && (cudaGetLastError() != cudaSuccess || cyc <= 0)) return DD_ERR_CUDA;
    // per iteration a thread performs 8 channels x 2 DM trials x 33 adds
    if (rc == DD_OK) *out = 512.0 * 256 * 8 * 2 * 33 / cyc;
    return rc;
}

#endif  // DD_TUNING

// SM clock under load: cycles of a long lane-rate launch against its CUDA-event time
int sm_clock_mhz(Scratch &s, double *out)
{
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return DD_ERR_CUDA;
    lane_rate_kernel<DD_PROBE_IMAD><<<s.nsm, kThreads>>>(s.sink, s.cycles, 1u);
    cudaEventRecord(e0);
    for (int r = 0; r < 8; ++r) lane_rate_kernel<DD_PROBE_IMAD><<<s.nsm, kThreads>>>(s.sink, s.cycles, 1u);
    cudaEventRecord(e1);
    int rc = DD_OK;
    float ms = 0.f;
    if (cudaEventSynchronize(e1) != cudaSuccess || cudaEventElapsedTime(&ms, e0, e1) != cudaSuccess) rc = DD_ERR_CUDA;
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (rc != DD_OK) return rc;
    std::vector<long long> h(static_cast<size_t>(s.nsm));
    if (cudaMemcpy(h.data(), s.cycles, h.size() * sizeof(long long), cudaMemcpyDeviceToHost) != cudaSuccess)
        return DD_ERR_CUDA;
    std::nth_element(h.begin(), h.begin() + h.size() / 2, h.end());
    // 8 back-to-back launches; the in-kernel loop is all but a few microseconds of each
    *out = 8.0 * static_cast<double>(h[h.size() / 2]) / (static_cast<double>(ms) * 1e3);
    return DD_OK;
}

}  // namespace

extern "C" int dd_probe(int what, double *value)
{
    if (!value) return DD_ERR_INVALID_ARG;
    int dev = -1;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) {
        cudaGetLastError();
        return DD_ERR_CUDA;
    }
    if (prop.major != 10) return DD_ERR_UNSUPPORTED_DEVICE;
    if (what == DD_PROBE_SM_COUNT) {
        *value = prop.multiProcessorCount;
        return DD_OK;
    }
    Scratch s;
    s.nsm = prop.multiProcessorCount;
    if (cudaMalloc(reinterpret_cast<void **>(&s.sink), static_cast<size_t>(s.nsm) * kThreads * 4) != cudaSuccess ||
        cudaMalloc(reinterpret_cast<void **>(&s.cycles), static_cast<size_t>(s.nsm) * sizeof(long long)) != cudaSuccess) {
        cudaGetLastError();
        return DD_ERR_ALLOC;
    }
    if (cudaMemset(s.sink, 0x5A, static_cast<size_t>(s.nsm) * kThreads * 4) != cudaSuccess) return DD_ERR_CUDA;
    switch (what) {
    case DD_PROBE_SM_CLOCK_MHZ: return sm_clock_mhz(s, value);
    case DD_PROBE_LDS32: return lds_rate<1>(s, value);
    case DD_PROBE_LDS64: return lds_rate<2>(s, value);
    case DD_PROBE_LDS128: return lds_rate<4>(s, value);
    case DD_PROBE_IADD3: return lane_rate<DD_PROBE_IADD3>(s, value);
    case DD_PROBE_VIADD16X2: return lane_rate<DD_PROBE_VIADD16X2>(s, value);
    case DD_PROBE_IMAD: return lane_rate<DD_PROBE_IMAD>(s, value);
    case DD_PROBE_FADD: return lane_rate<DD_PROBE_FADD>(s, value);
    case DD_PROBE_LOP3: return lane_rate<DD_PROBE_LOP3>(s, value);
    case DD_PROBE_PRMT: return lane_rate<DD_PROBE_PRMT>(s, value);
    case DD_PROBE_SHIFT_ADD: return lane_rate<DD_PROBE_SHIFT_ADD>(s, value);
    case DD_PROBE_IMAD_HI: return lane_rate<DD_PROBE_IMAD_HI>(s, value);
    case DD_PROBE_IDP4A: return lane_rate<DD_PROBE_IDP4A>(s, value);
    case DD_PROBE_SHF: return lane_rate<DD_PROBE_SHF>(s, value);
#ifdef DD_TUNING
    case DD_PROBE_TMEM_LD: return tmem_rate<0>(s, value);
    case DD_PROBE_TMEM_LD_WITH_LDS: return tmem_rate<1>(s, value);
    case DD_PROBE_F32_ADDS_SMEM_ONLY: return hybrid_rate<0, true>(s, value);
    case DD_PROBE_F32_ADDS_TMEM_4_OF_8: return hybrid_rate<4, true>(s, value);
    case DD_PROBE_F32_ADDS_TMEM_4_OF_8_NO_FILL: return hybrid_rate<4, false>(s, value);
#endif
    default: return DD_ERR_INVALID_ARG;
    }
}
