// dd_kernels.cu -- sm_100a kernels of libdd.so.
//
// Two kernels per dd_execute:
//   1. interleave_kernel: in[c][t] (u8/u16/f32) -> X[c][j] (32-bit words), lane k of word j
//      holding in[c][k*L + j].  HBM-bound, ~2x the input size of traffic.
//   2. dedisperse_kernel: the shifted sum.  A thread block owns D_DM DM trials x D_J words of
//      the interleaved time axis.  A producer warp streams channel rows into a ring of
//      shared-memory stages with cp.async.bulk (TMA 1-D, mbarrier complete_tx); consumer
//      warps read one 32-bit word per lane at the (DM, channel) word offset -- conflict-free
//      for ANY shift -- and accumulate LANES samples per word:
//        u8 : W += w (carries run across byte lanes), O += odd bytes of w as two 16-bit
//             lanes (PRMT); even lanes are recovered as W - 256*O at the flush, every
//             256 channels (exact: 257*255 < 2^16), into four uint32 accumulators;
//        u16: W += w, H += w >> 16; low lane recovered as W - 65536*H at the end;
//        f32: FADD.
// No tensor cores: a shifted-diagonal sum is not a contraction.
#include <cuda_runtime.h>

#include <cstdint>

#include "dd_internal.h"

namespace dd {
namespace {

// ------------------------------------------------------------------ PTX helpers
__device__ __forceinline__ uint32_t smem_u32(const void *p)
{
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "WAIT_LOOP:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra.uni WAIT_DONE;\n\t"
        "bra.uni WAIT_LOOP;\n\t"
        "WAIT_DONE:\n\t"
        "}" ::"r"(bar),
        "r"(parity)
        : "memory");
}
// 1-D bulk copy global -> shared, completion counted in bytes on an mbarrier (SASS: UBLKCP).
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar)
{
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
        "l"(src), "r"(bytes), "r"(bar)
        : "memory");
}
__device__ __forceinline__ uint32_t odd_bytes(uint32_t w)
{
    // bytes 1 and 3 of w as two 16-bit lanes: one PRMT
    return __byte_perm(w, 0u, 0x4341);
}

// ------------------------------------------------------------------ per-mode accumulators
template <int MODE>
struct Acc;

template <>
struct Acc<DD_U8> {
    uint32_t W = 0, O = 0;           // packed, flushed every <= 256 channels
    uint32_t a0 = 0, a1 = 0, a2 = 0, a3 = 0;
    __device__ __forceinline__ void add2(uint32_t x, uint32_t y)
    {
        W = W + x + y;
        O = O + odd_bytes(x) + odd_bytes(y);
    }
    __device__ __forceinline__ void flush()
    {
        const uint32_t E = W - (O << 8);
        a0 += E & 0xFFFFu;
        a2 += E >> 16;
        a1 += O & 0xFFFFu;
        a3 += O >> 16;
        W = 0;
        O = 0;
    }
    static constexpr bool kNeedsFlush = true;
};

template <>
struct Acc<DD_U16> {
    uint32_t W = 0, H = 0;
    __device__ __forceinline__ void add2(uint32_t x, uint32_t y)
    {
        W = W + x + y;
        H = H + (x >> 16) + (y >> 16);
    }
    __device__ __forceinline__ void flush() {}
    static constexpr bool kNeedsFlush = false;
};

template <>
struct Acc<DD_F32> {
    float s = 0.f;
    __device__ __forceinline__ void add2(uint32_t x, uint32_t y)
    {
        s += __uint_as_float(x);
        s += __uint_as_float(y);
    }
    __device__ __forceinline__ void flush() {}
    static constexpr bool kNeedsFlush = false;
};

// ------------------------------------------------------------------ main kernel
template <int MODE, int RD, int RW, int WD, int WJ, int CH>
__global__ void __launch_bounds__((WD * WJ + 1) * 32, 1) dedisperse_kernel(const KernelParams p)
{
    constexpr int NCW = WD * WJ;  // consumer warps
    constexpr int D_DM = RD * WD;
    constexpr int D_J = RW * WJ * 32;
    constexpr int LANES = MODE == DD_U8 ? 4 : (MODE == DD_U16 ? 2 : 1);
    static_assert(CH % 4 == 0 && CH <= 32, "CH: multiple of 4, one producer lane per channel");
    static_assert(256 % CH == 0, "u8 flush period must be a whole number of stages");

    extern __shared__ __align__(128) unsigned char smem[];
    // [0, 1024): mbarriers full[nstage], empty[nstage]; then nstage stage buffers, each
    // CH rows of pitch_bytes followed by the D_DM x CH int32 offset table.
    const uint32_t bar_full = smem_u32(smem);
    const uint32_t bar_empty = bar_full + 8u * 8u;
    unsigned char *stage0 = smem + 1024;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int b = blockIdx.x % p.ndb;  // DM block fastest: co-resident blocks share input
    const int jt = blockIdx.x / p.ndb;
    const int64_t j0 = static_cast<int64_t>(jt) * D_J;
    const int nstage = p.nstage;

    if (threadIdx.x == 0) {
        for (int s = 0; s < nstage; ++s) {
            mbar_init(bar_full + 8u * s, 1);
            mbar_init(bar_empty + 8u * s, NCW);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp == NCW) {
        // ===================== producer warp: lane l stages channel l of each stage
        const int32_t *base_row = p.blk_base + static_cast<size_t>(b) * p.nch_pad;
        const int32_t *len_row = p.blk_len + static_cast<size_t>(b) * p.nch_pad;
        const int32_t *ofs_blk = p.ofs + static_cast<size_t>(b) * p.nk * (D_DM * CH);
        int s = 0;
        uint32_t phase = 0;
        for (int k = 0; k < p.nk; ++k) {
            uint32_t bytes = 0;
            const uint32_t *src = nullptr;
            if (lane < CH) {
                const int c = k * CH + lane;
                bytes = static_cast<uint32_t>(len_row[c]);
                src = p.X + static_cast<size_t>(c) * p.Lw + j0 + base_row[c];
            }
            const uint32_t total = __reduce_add_sync(0xffffffffu, bytes) + D_DM * CH * 4;
            if (k >= nstage) mbar_wait(bar_empty + 8u * s, phase ^ 1u);
            const uint32_t full = bar_full + 8u * s;
            const uint32_t dst = smem_u32(stage0) + static_cast<uint32_t>(s) * p.stage_bytes;
            if (lane == 0) {
                mbar_arrive_expect_tx(full, total);
                bulk_g2s(dst + CH * p.pitch_bytes, ofs_blk + static_cast<size_t>(k) * (D_DM * CH),
                         D_DM * CH * 4, full);
            }
            __syncwarp();
            if (lane < CH) bulk_g2s(dst + lane * p.pitch_bytes, src, bytes, full);
            if (++s == nstage) {
                s = 0;
                phase ^= 1u;
            }
        }
        return;
    }

    // ========================= consumer warps
    const int wd = warp / WJ, wj = warp % WJ;
    Acc<MODE> acc[RD][RW];
    const uint32_t lane_byte = static_cast<uint32_t>((wj * RW * 32 + lane) * 4);

    int s = 0;
    uint32_t phase = 0;
    for (int k = 0; k < p.nk; ++k) {
        mbar_wait(bar_full + 8u * s, phase);
        const unsigned char *stage = stage0 + static_cast<size_t>(s) * p.stage_bytes;
        const unsigned char *rows = stage + lane_byte;
        const int4 *otab = reinterpret_cast<const int4 *>(stage + CH * p.pitch_bytes) +
                           (wd * RD) * (CH / 4);
#pragma unroll
        for (int c4 = 0; c4 < CH / 4; ++c4) {
            int4 o[RD];
#pragma unroll
            for (int r = 0; r < RD; ++r) o[r] = otab[r * (CH / 4) + c4];
#pragma unroll
            for (int r = 0; r < RD; ++r) {
                const uint32_t *q0 = reinterpret_cast<const uint32_t *>(rows + o[r].x);
                const uint32_t *q1 = reinterpret_cast<const uint32_t *>(rows + o[r].y);
                const uint32_t *q2 = reinterpret_cast<const uint32_t *>(rows + o[r].z);
                const uint32_t *q3 = reinterpret_cast<const uint32_t *>(rows + o[r].w);
#pragma unroll
                for (int i = 0; i < RW; ++i) acc[r][i].add2(q0[i * 32], q1[i * 32]);
#pragma unroll
                for (int i = 0; i < RW; ++i) acc[r][i].add2(q2[i * 32], q3[i * 32]);
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_empty + 8u * s);
        if (Acc<MODE>::kNeedsFlush && (((k + 1) * CH) & 255) == 0) {
#pragma unroll
            for (int r = 0; r < RD; ++r)
#pragma unroll
                for (int i = 0; i < RW; ++i) acc[r][i].flush();
        }
        if (++s == nstage) {
            s = 0;
            phase ^= 1u;
        }
    }

    // ========================= store (a7): lane k of word j is output sample k*L + j
#pragma unroll
    for (int r = 0; r < RD; ++r) {
        const int d = b * D_DM + wd * RD + r;
        if (d >= p.ndm) continue;
#pragma unroll
        for (int i = 0; i < RW; ++i) {
            const int64_t j = j0 + (wj * RW + i) * 32 + lane;
            if (j >= p.L) continue;
            if constexpr (MODE == DD_U8) {
                Acc<DD_U8> &a = acc[r][i];
                a.flush();
                uint32_t *o = static_cast<uint32_t *>(p.out) + static_cast<size_t>(d) * p.out_len;
                const uint32_t v[4] = {a.a0, a.a1, a.a2, a.a3};
#pragma unroll
                for (int l = 0; l < LANES; ++l) {
                    const int64_t t = l * p.L + j;
                    if (t < p.out_len) o[t] = v[l];
                }
            } else if constexpr (MODE == DD_U16) {
                Acc<DD_U16> &a = acc[r][i];
                uint32_t *o = static_cast<uint32_t *>(p.out) + static_cast<size_t>(d) * p.out_len;
                const uint32_t v[2] = {a.W - (a.H << 16), a.H};
#pragma unroll
                for (int l = 0; l < LANES; ++l) {
                    const int64_t t = l * p.L + j;
                    if (t < p.out_len) o[t] = v[l];
                }
            } else {
                Acc<DD_F32> &a = acc[r][i];
                float *o = static_cast<float *>(p.out) + static_cast<size_t>(d) * p.out_len;
                if (j < p.out_len) o[j] = a.s;
            }
        }
    }
}

// ------------------------------------------------------------------ interleave pre-pass
// One thread makes four consecutive words (one 16-byte store).  Reads past the end of a
// row (t >= nsamps) give 0; such lanes only feed outputs that are never stored.
template <typename T>
__device__ __forceinline__ uint32_t sample_or_zero(const T *row, int64_t t, int64_t nsamps)
{
    return t < nsamps ? static_cast<uint32_t>(row[t]) : 0u;
}

template <int MODE>
__global__ void __launch_bounds__(256) interleave_kernel(const InterleaveParams p)
{
    const int c = static_cast<int>(blockIdx.x / p.nchunk);
    const int64_t j = (static_cast<int64_t>(blockIdx.x % p.nchunk) * blockDim.x + threadIdx.x) * 4;
    if (j >= p.Lw) return;
    uint4 w;
    if (MODE == DD_U8) {
        const uint8_t *row = static_cast<const uint8_t *>(p.in) + static_cast<size_t>(c) * p.nsamps;
        const bool aligned = (reinterpret_cast<uintptr_t>(row) & 3u) == 0;
        uint32_t seg[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const int64_t t = k * p.L + j;
            if (aligned && t + 3 < p.nsamps) {
                seg[k] = *reinterpret_cast<const uint32_t *>(row + t);
            } else {
                seg[k] = sample_or_zero(row, t, p.nsamps) | sample_or_zero(row, t + 1, p.nsamps) << 8 |
                         sample_or_zero(row, t + 2, p.nsamps) << 16 |
                         sample_or_zero(row, t + 3, p.nsamps) << 24;
            }
        }
        // 4x4 byte transpose: word n gets byte n of each segment
        const uint32_t t01l = __byte_perm(seg[0], seg[1], 0x5140);  // a0 b0 a1 b1
        const uint32_t t01h = __byte_perm(seg[0], seg[1], 0x7362);  // a2 b2 a3 b3
        const uint32_t t23l = __byte_perm(seg[2], seg[3], 0x5140);
        const uint32_t t23h = __byte_perm(seg[2], seg[3], 0x7362);
        w.x = __byte_perm(t01l, t23l, 0x5410);
        w.y = __byte_perm(t01l, t23l, 0x7632);
        w.z = __byte_perm(t01h, t23h, 0x5410);
        w.w = __byte_perm(t01h, t23h, 0x7632);
    } else if (MODE == DD_U16) {
        const uint16_t *row = static_cast<const uint16_t *>(p.in) + static_cast<size_t>(c) * p.nsamps;
        const bool aligned = (reinterpret_cast<uintptr_t>(row) & 7u) == 0;
        uint2 seg[2];
#pragma unroll
        for (int k = 0; k < 2; ++k) {
            const int64_t t = k * p.L + j;
            if (aligned && t + 3 < p.nsamps) {
                seg[k] = *reinterpret_cast<const uint2 *>(row + t);
            } else {
                seg[k].x = sample_or_zero(row, t, p.nsamps) | sample_or_zero(row, t + 1, p.nsamps) << 16;
                seg[k].y = sample_or_zero(row, t + 2, p.nsamps) | sample_or_zero(row, t + 3, p.nsamps) << 16;
            }
        }
        w.x = __byte_perm(seg[0].x, seg[1].x, 0x5410);
        w.y = __byte_perm(seg[0].x, seg[1].x, 0x7632);
        w.z = __byte_perm(seg[0].y, seg[1].y, 0x5410);
        w.w = __byte_perm(seg[0].y, seg[1].y, 0x7632);
    } else {
        const uint32_t *row = static_cast<const uint32_t *>(p.in) + static_cast<size_t>(c) * p.nsamps;
        const bool aligned = (reinterpret_cast<uintptr_t>(row) & 15u) == 0;
        if (aligned && j + 3 < p.nsamps) {
            w = *reinterpret_cast<const uint4 *>(row + j);
        } else {
            w.x = sample_or_zero(row, j, p.nsamps);
            w.y = sample_or_zero(row, j + 1, p.nsamps);
            w.z = sample_or_zero(row, j + 2, p.nsamps);
            w.w = sample_or_zero(row, j + 3, p.nsamps);
        }
    }
    *reinterpret_cast<uint4 *>(p.X + static_cast<size_t>(c) * p.Lw + j) = w;
}

// ------------------------------------------------------------------ variant table
using KernelFn = void (*)(const KernelParams);
struct Variant {
    KernelShape shape;
    KernelFn fn;
};

#define DD_VARIANT(MODE, LANES, RD, RW, WD, WJ, CH)               \
    {                                                             \
        {MODE, LANES, RD, RW, WD, WJ, CH}, dedisperse_kernel<MODE, RD, RW, WD, WJ, CH> \
    }

// Ordered per mode from the largest DM block to the smallest; dd_plan_create takes the
// first whose shared-memory ring fits (smaller DM blocks = shorter staged windows).
const Variant kVariants[] = {
    DD_VARIANT(DD_U8, 4, 1, 8, 16, 1, 16),
    DD_VARIANT(DD_U8, 4, 1, 8, 8, 2, 16),
    DD_VARIANT(DD_U8, 4, 1, 8, 4, 4, 16),
    DD_VARIANT(DD_U8, 4, 1, 8, 1, 16, 16),
    DD_VARIANT(DD_U16, 2, 2, 8, 16, 1, 16),
    DD_VARIANT(DD_U16, 2, 1, 8, 16, 1, 16),
    DD_VARIANT(DD_U16, 2, 1, 8, 4, 4, 16),
    DD_VARIANT(DD_U16, 2, 1, 8, 1, 16, 16),
    DD_VARIANT(DD_F32, 1, 2, 8, 16, 1, 16),
    DD_VARIANT(DD_F32, 1, 1, 8, 16, 1, 16),
    DD_VARIANT(DD_F32, 1, 1, 8, 4, 4, 16),
    DD_VARIANT(DD_F32, 1, 1, 8, 1, 16, 16),
};
constexpr int kNumVariants = sizeof(kVariants) / sizeof(kVariants[0]);

}  // namespace

int num_variants() { return kNumVariants; }
const KernelShape &variant_shape(int v) { return kVariants[v].shape; }

int variant_prepare(int v, int smem_bytes)
{
    return static_cast<int>(cudaFuncSetAttribute(reinterpret_cast<const void *>(kVariants[v].fn),
                                                 cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                 smem_bytes));
}

int launch_dedisperse(int v, const KernelParams &p, int grid, int smem_bytes, void *stream)
{
    const Variant &var = kVariants[v];
    var.fn<<<grid, var.shape.threads(), smem_bytes, static_cast<cudaStream_t>(stream)>>>(p);
    return static_cast<int>(cudaGetLastError());
}

int launch_interleave(int mode, const InterleaveParams &p, void *stream)
{
    const unsigned grid = static_cast<unsigned>(static_cast<int64_t>(p.nchunk) * p.nchans);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (mode == DD_U8)
        interleave_kernel<DD_U8><<<grid, 256, 0, st>>>(p);
    else if (mode == DD_U16)
        interleave_kernel<DD_U16><<<grid, 256, 0, st>>>(p);
    else
        interleave_kernel<DD_F32><<<grid, 256, 0, st>>>(p);
    return static_cast<int>(cudaGetLastError());
}

}  // namespace dd
