// dd_kernels.cu -- sm_100a kernels of libdd.so.
//
// Two kernels per dd_execute:
//   1. interleave_kernel (interleave_tm_kernel for time-major input): in[c][t] (u4/u8/u16/f32)
//      -> X[c][j], superwords of VW 32-bit words, lane l of superword j holding in[c][l*L + j].
//      HBM-bound.
//   2. dedisperse_kernel: the shifted sum.  A thread block owns D_DM DM trials x D_J
//      superwords of the interleaved time axis.  A producer warp streams channel windows into
//      a ring of shared-memory stages with cp.async.bulk (TMA 1-D, mbarrier complete_tx);
//      consumer warps read one superword per lane (LDS.32/64/128) at the (DM, channel) offset
//      -- aligned and conflict-free for ANY shift -- and accumulate all its lanes at once:
//        u8 : W += w (carries run across byte lanes), O += odd bytes of w as two 16-bit
//             lanes (PRMT, the add as IMAD on the fma pipe); even lanes are recovered as
//             W - 256*O at the flush, after at most 256 channels (256*255 < 2^16), into four
//             uint32 accumulators per word that live in tensor memory (lane-private scratch);
//        u16: W += w, H += w >> 16; low lane recovered as W - 65536*H at the end;
//        u4 : eight 4-bit lanes per word stay packed in shared memory (0.5 B per add): W += w
//             (carries run across nibble lanes), A += odd nibbles of w as byte lanes (LOP3 + LEA.HI);
//             per stage the byte lanes fold into 16-bit lanes, every <= 4096 channels into uint32
//             accumulators in tensor memory;
//        f32: FADD.
//      The grid is rasterised in DM-block panels so that a wave's input footprint is streamed
//      from HBM once (tile_of_cta).
// Also here: interleave_u4_kernel / interleave_tm_u4_kernel (4-bit pre-passes), transpose_kernel and
// transpose_u4_kernel (dd_transpose), bin_time_*_kernel (dd_bin_time).
// The tensor cores' MMA units are not used: a shifted-diagonal sum is not a contraction.
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

// ------------------------------------------------------------------ tensor-memory scratch (FM = 4)
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&r)[16])
{
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
          "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
        : "r"(taddr)
        : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t (&r)[16])
{
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};"
        :
        : "r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]),
          "r"(r[8]), "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15])
        : "memory");
}

// ------------------------------------------------------------------ per-mode accumulators
template <int MODE, int FM>
struct Acc;

// FM (u8 only) = which adds are issued as IMAD (x * one + acc, `one` a runtime 1 that ptxas
// cannot fold) on the fma pipe instead of IADD3 on the alu pipe:
//   0 none; 1 W += x (both words); 2 O += odd(x) (both words);
//   4 = 2, and the four uint32 flush accumulators per word live in tensor memory instead of
//       registers (TMEM is lane-private scratch here: a thread reads and writes only its own lane)
template <int FM>
struct Acc<DD_U8, FM> {
    uint32_t W = 0, O = 0;           // packed, flushed every <= 256 channels
    uint32_t a0 = 0, a1 = 0, a2 = 0, a3 = 0;
    __device__ __forceinline__ void add2(uint32_t x, uint32_t y, uint32_t one)
    {
        if (FM == 1) {
            W = x * one + W;
            W = y * one + W;
        } else {
            W = W + x + y;
        }
        if (FM == 2 || FM == 4) {
            O = odd_bytes(x) * one + O;
            O = odd_bytes(y) * one + O;
        } else {
            O = O + odd_bytes(x) + odd_bytes(y);
        }
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
    // the four lane sums held in the packed accumulators, which are then cleared
    __device__ __forceinline__ void drain(uint32_t (&v)[4])
    {
        const uint32_t E = W - (O << 8);
        v[0] = E & 0xFFFFu;
        v[1] = O & 0xFFFFu;
        v[2] = E >> 16;
        v[3] = O >> 16;
        W = 0;
        O = 0;
    }
    static constexpr bool kNeedsFlush = true;
};

// Packed 4-bit samples, eight per 32-bit word (nibble n of a word = lane n).  Three levels:
//   1. per stage (<= 16 channels; 17 * 15 = 255): W += x on the whole word (carries run across
//      nibble lanes) and A += odd nibbles of x as four byte lanes (one LOP3 + one shift-and-add,
//      SASS LEA.HI); the even nibbles are recovered exactly as byte lanes E = W - 16*A.
//   2. at the end of every stage E and A are added into 16-bit lanes with the 8-bit trick
//      (We += E, Oe += odd bytes of E; Wa += A, Oa += odd bytes of A): good for 4369 channels.
//   3. every <= 4096 channels the eight 16-bit lanes of a word go to eight uint32 accumulators in
//      tensor memory (lane-private scratch, as for 8-bit).
// FM: 0 = W on the fma pipe (IMAD), the shift-and-add on the alu pipe; 1 = W as IADD3 as well;
//     2 = shift and mask (SHF + LOP3) on the alu pipe, both adds as IMAD on the fma pipe
template <int FM>
struct Acc<DD_U4, FM> {
    uint32_t W = 0, A = 0, Whi = 0;
    uint32_t We = 0, Oe = 0, Wa = 0, Oa = 0;
    static __device__ __forceinline__ uint32_t oddn(uint32_t x)
    {
        if (FM == 2) return (x >> 4) & 0x0F0F0F0Fu;
        return (x & 0xF0F0F0F0u) >> 4;
    }
    static __device__ __forceinline__ void lea_add(uint32_t &a, uint32_t x)
    {
        asm("{ .reg .u32 t; and.b32 t, %1, 0xF0F0F0F0; shr.u32 t, t, 4; add.u32 %0, %0, t; }" : "+r"(a) : "r"(x));
    }
    static __device__ __forceinline__ void wide_add(uint32_t &lo, uint32_t &hi, uint32_t x, uint32_t one)
    {
        asm("{ .reg .u64 w; mov.b64 w, {%0, %1}; mad.wide.u32 w, %2, %3, w; mov.b64 {%0, %1}, w; }"
            : "+r"(lo), "+r"(hi)
            : "r"(x), "r"(one));
    }
    // first channel pair of a stage: overwrite the level-1 accumulators
    __device__ __forceinline__ void set2(uint32_t x, uint32_t y, uint32_t one)
    {
        if (FM == 3) {  // A = even nibbles as byte lanes, (Whi:W) = exact 64-bit sum of the words
            A = (x & 0x0F0F0F0Fu) + (y & 0x0F0F0F0Fu);
            W = x;
            Whi = 0u;
            wide_add(W, Whi, y, one);
        } else if (FM == 1) {
            W = x + y;
            A = oddn(x) + oddn(y);
        } else if (FM == 2) {
            W = y * one + x;
            A = oddn(y) * one + oddn(x);
        } else if (FM == 4) {
            W = y * one + x;
            A = oddn(x);
            lea_add(A, y);
        } else {
            W = y * one + x;
            A = oddn(x) + oddn(y);
        }
    }
    __device__ __forceinline__ void add2(uint32_t x, uint32_t y, uint32_t one)
    {
        if (FM == 3) {
            A = A + (x & 0x0F0F0F0Fu) + (y & 0x0F0F0F0Fu);
            wide_add(W, Whi, x, one);
            wide_add(W, Whi, y, one);
        } else if (FM == 1) {
            W = W + x + y;
            A = A + oddn(x);
            A = A + oddn(y);
        } else if (FM == 2) {
            W = x * one + W;
            W = y * one + W;
            A = oddn(x) * one + A;
            A = oddn(y) * one + A;
        } else if (FM == 4) {
            W = x * one + W;
            W = y * one + W;
            lea_add(A, x);
            lea_add(A, y);
        } else {
            W = x * one + W;
            W = y * one + W;
            A = A + oddn(x);
            A = A + oddn(y);
        }
    }
    // end of a stage: level 1 -> level 2
    __device__ __forceinline__ void flush()
    {
        uint32_t E, O;
        if (FM == 3) {
            E = A;
            const uint64_t w = (static_cast<uint64_t>(Whi) << 32 | W) - A;  // 16 * (odd nibbles as byte lanes), < 2^36
            O = static_cast<uint32_t>(w >> 4);
        } else {
            E = W - (A << 4);
            O = A;
        }
        We += E;
        Oe += odd_bytes(E);
        Wa += O;
        Oa += odd_bytes(O);
    }
    // the eight lane sums held in level 2 (lane n = nibble n), which is then cleared
    __device__ __forceinline__ void drain(uint32_t (&v)[8])
    {
        const uint32_t E2 = We - (Oe << 8), A2 = Wa - (Oa << 8);
        v[0] = E2 & 0xFFFFu;
        v[1] = A2 & 0xFFFFu;
        v[2] = Oe & 0xFFFFu;
        v[3] = Oa & 0xFFFFu;
        v[4] = E2 >> 16;
        v[5] = A2 >> 16;
        v[6] = Oe >> 16;
        v[7] = Oa >> 16;
        We = Oe = Wa = Oa = 0u;
    }
    static constexpr bool kNeedsFlush = true;
};

template <int FM>
struct Acc<DD_U16, FM> {
    uint32_t W = 0, H = 0;
    __device__ __forceinline__ void add2(uint32_t x, uint32_t y, uint32_t)
    {
        W = W + x + y;
        H = H + (x >> 16) + (y >> 16);
    }
    __device__ __forceinline__ void flush() {}
    static constexpr bool kNeedsFlush = false;
};

template <int FM>
struct Acc<DD_F32, FM> {
    float s = 0.f;
    __device__ __forceinline__ void add2(uint32_t x, uint32_t y, uint32_t)
    {
        s += __uint_as_float(x);
        s += __uint_as_float(y);
    }
    __device__ __forceinline__ void flush() {}
    static constexpr bool kNeedsFlush = false;
};

// ------------------------------------------------------------------ main kernel
// One shared-memory load of VW words (LDS.32 / LDS.64 / LDS.128) at a 32-bit shared-space
// address plus a compile-time byte offset.
template <int VW>
struct SW;
template <>
struct SW<1> {
    uint32_t w[1];
    template <int IMM>
    __device__ __forceinline__ void load(uint32_t a)
    {
        asm volatile("ld.shared.u32 %0, [%1+%2];" : "=r"(w[0]) : "r"(a), "n"(IMM) : "memory");
    }
};
template <>
struct SW<2> {
    uint32_t w[2];
    template <int IMM>
    __device__ __forceinline__ void load(uint32_t a)
    {
        asm volatile("ld.shared.v2.u32 {%0,%1}, [%2+%3];" : "=r"(w[0]), "=r"(w[1]) : "r"(a), "n"(IMM) : "memory");
    }
};
template <>
struct SW<4> {
    uint32_t w[4];
    template <int IMM>
    __device__ __forceinline__ void load(uint32_t a)
    {
        asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4+%5];"
                     : "=r"(w[0]), "=r"(w[1]), "=r"(w[2]), "=r"(w[3])
                     : "r"(a), "n"(IMM)
                     : "memory");
    }
};

// RJ superword loads of one channel row (stride 32 superwords) added into acc[.][.].
template <int MODE, int VW, int RJ, int FM, int I = 0>
struct RowPair {
    // first: the first channel pair of a stage (4-bit: the per-stage accumulators are overwritten)
    static __device__ __forceinline__ void run(Acc<MODE, FM> (&acc)[RJ][VW], uint32_t a0, uint32_t a1,
                                               uint32_t one, bool first)
    {
        SW<VW> x, y;
        x.template load<I * 32 * VW * 4>(a0);
        y.template load<I * 32 * VW * 4>(a1);
#pragma unroll
        for (int v = 0; v < VW; ++v) {
            if constexpr (MODE == DD_U4) {
                if (first)
                    acc[I][v].set2(x.w[v], y.w[v], one);
                else
                    acc[I][v].add2(x.w[v], y.w[v], one);
            } else {
                acc[I][v].add2(x.w[v], y.w[v], one);
            }
        }
        RowPair<MODE, VW, RJ, FM, I + 1>::run(acc, a0, a1, one, first);
    }
};
template <int MODE, int VW, int RJ, int FM>
struct RowPair<MODE, VW, RJ, FM, RJ> {
    static __device__ __forceinline__ void run(Acc<MODE, FM> (&)[RJ][VW], uint32_t, uint32_t, uint32_t, bool) {}
};

// Rasterisation of the main kernel's grid: DM blocks are grouped in panels of p.panel; inside a
// panel the DM block runs fastest, then the j tile.  The CTAs resident at one time (one wave)
// then cover ~panel DM blocks x (SMs / panel) j tiles, the shape that minimises the input
// footprint of a wave -- every wave streams its footprint from HBM once (DESIGN.md "DRAM
// traffic").  Returns the DM block and the j tile of CTA `bid`.
__device__ __forceinline__ void tile_of_cta(const KernelParams &p, int bid, int &b, int &jt)
{
    const int per_panel = p.panel * p.ntj;
    const int pn = bid / per_panel;
    const int rem = bid - pn * per_panel;
    const int nb = min(p.panel, p.ndb - pn * p.panel);
    b = pn * p.panel + rem % nb;
    jt = rem / nb + p.jt_begin;
}

template <int MODE, int VW, int RD, int RJ, int WD, int WJ, int CH, int FM, int NB, int OW>
__global__ void __launch_bounds__((WD * WJ + 1) * 32, NB) dedisperse_kernel(const KernelParams p)
{
    constexpr int NCW = WD * WJ;  // consumer warps
    constexpr int D_DM = RD * WD;
    constexpr int D_J = RJ * WJ * 32;  // superwords
    constexpr int S = VW * 4;          // bytes per superword
    constexpr int LPW = MODE == DD_U4 ? 8 : (MODE == DD_U8 ? 4 : (MODE == DD_U16 ? 2 : 1));  // samples per word
    static_assert(CH % (16 / OW) == 0 && CH <= 32, "CH: whole LDS.128 offset loads, one producer lane per channel");

    extern __shared__ __align__(128) unsigned char smem[];
    // [0, 1024): mbarriers full[nstage], empty[nstage]; then nstage stage buffers, each the
    // packed channel windows (rows_bytes) followed by the D_DM x CH offset table (OW = 4: byte offsets; OW = 2: uint16 in units of 4 bytes).
    const uint32_t bar_full = smem_u32(smem);
    const uint32_t bar_empty = bar_full + 8u * 8u;
    unsigned char *stage0 = smem + 1024;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int nstage = p.nstage;

    if (threadIdx.x == 0) {
        for (int s = 0; s < nstage; ++s) {
            mbar_init(bar_full + 8u * s, 1);
            mbar_init(bar_empty + 8u * s, NCW);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    constexpr bool TMEM = (MODE == DD_U8 && FM == 4) || MODE == DD_U4;
    constexpr int NCOL = LPW * RD * RJ * VW;  // TMEM columns per consumer thread (one uint32 per lane of a word)
    constexpr int WPC = 16 / LPW;             // words per 16-column tcgen05.ld / st
    // channels between two flushes to the uint32 accumulators (16-bit lanes: 256 * 255, 4096 * 15 < 2^16)
    constexpr int FLUSH_CH = MODE == DD_U4 ? 4096 : 256;
    static_assert(MODE != DD_U4 || CH <= 16, "4-bit: a stage's byte lanes hold at most 17 channels");
    static_assert(!TMEM || (NCOL % 16 == 0 && (NCW + 3) / 4 * NCOL <= 512), "TMEM scratch layout");
    // columns this shape needs, rounded up to the power of two >= 32 that tcgen05.alloc takes
    constexpr int TNEED = (NCW + 3) / 4 * NCOL;
    constexpr uint32_t TCOLS = TNEED <= 32 ? 32 : TNEED <= 64 ? 64 : TNEED <= 128 ? 128 : TNEED <= 256 ? 256 : 512;
    if (TMEM && warp == 0) {  // one warp allocates (blocks until a co-resident TMEM user frees enough)
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(bar_full + 960u), "n"(TCOLS) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    __syncthreads();
    if (TMEM) asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");

    if (warp == NCW) {
        // ===================== producer warp: lane l stages slot l of each stage
        int b, jt;
        tile_of_cta(p, blockIdx.x, b, jt);
        const int64_t j0 = static_cast<int64_t>(jt) * D_J;
        const int4 *blk = reinterpret_cast<const int4 *>(p.blk) + static_cast<size_t>(b) * p.nch_pad;
        const unsigned char *ofs_blk =
            static_cast<const unsigned char *>(p.ofs) + static_cast<size_t>(b) * p.nk * (D_DM * CH * OW);
        const unsigned char *Xb = reinterpret_cast<const unsigned char *>(p.X);
        int s = 0;
        uint32_t phase = 0;
        int4 q = make_int4(0, 0, 0, 0);
        if (lane < CH) q = blk[lane];
        for (int k = 0; k < p.nk; ++k) {
            const uint32_t bytes = static_cast<uint32_t>(q.z);
            const unsigned char *src =
                Xb + (static_cast<size_t>(q.x) * p.Lw + j0 + q.y) * S;
            const uint32_t dsto = static_cast<uint32_t>(q.w);
            if (k + 1 < p.nk && lane < CH) q = blk[(k + 1) * CH + lane];  // prefetch next stage's slots
            const uint32_t total = __reduce_add_sync(0xffffffffu, bytes) + D_DM * CH * OW;
            if (k >= nstage) mbar_wait(bar_empty + 8u * s, phase ^ 1u);
            const uint32_t full = bar_full + 8u * s;
            const uint32_t dst = smem_u32(stage0) + static_cast<uint32_t>(s) * p.stage_bytes;
            if (lane == 0) {
                mbar_arrive_expect_tx(full, total);
                bulk_g2s(dst + p.rows_bytes, ofs_blk + static_cast<size_t>(k) * (D_DM * CH * OW),
                         D_DM * CH * OW, full);
            }
            __syncwarp();
            if (lane < CH) bulk_g2s(dst + dsto, src, bytes, full);
            if (++s == nstage) {
                s = 0;
                phase ^= 1u;
            }
        }
        if (TMEM) asm volatile("bar.sync 1, %0;" ::"r"((NCW + 1) * 32) : "memory");  // TMEM is freed after the consumers
        return;
    }

    // ========================= consumer warps
    const int wd = warp / WJ, wj = warp % WJ;
    Acc<MODE, FM> acc[RD][RJ][VW];
    const uint32_t one = p.one;
    const uint32_t four = one * 4u;
    const uint32_t lane_byte = static_cast<uint32_t>((wj * RJ * 32 + lane) * S);
    const uint32_t stage_u32 = smem_u32(stage0);

    // FM = 4: this thread's 4 uint32 accumulators per word sit in its own TMEM lane, columns
    // [(warp / 4) * NCOL, +NCOL) of lane quarter warp % 4 (the hardware's rule: warp w of a CTA
    // reaches lanes 32 * (w % 4) .. +31); column ((r*RJ + i)*VW + v)*4 + l.  Touched only at a
    // flush (every 256 channels) and at the end, 16 columns per instruction.
    // (the address is re-read from shared memory at each of its rare uses: the hot loop is at the
    // register limit)
    auto tmem_addr = [&]() {
        uint32_t base;
        asm volatile("ld.shared.u32 %0, [%1];" : "=r"(base) : "r"(bar_full + 960u) : "memory");
        return base + (static_cast<uint32_t>((warp & 3) * 32) << 16) + static_cast<uint32_t>((warp >> 2) * NCOL);
    };
    bool parked = false;  // TMEM holds valid partial sums
    int s = 0;
    int since_flush = 0;
    uint32_t phase = 0;
    for (int k = 0; k < p.nk; ++k) {
        mbar_wait(bar_full + 8u * s, phase);
        const uint32_t stage = stage_u32 + static_cast<uint32_t>(s) * p.stage_bytes;
        const uint32_t rows = stage + lane_byte;
        const uint32_t otab = stage + p.rows_bytes + (wd * RD) * (CH * OW);
        // One LDS.128 fetches 16 / OW offsets per DM trial (a broadcast: the row is warp-uniform).
        // address = offset * scale + rows as IMAD on the fma pipe (`one` is opaque to ptxas).
        constexpr int NPER = 16 / OW;
#pragma unroll
        for (int cg = 0; cg < CH / NPER; ++cg) {
            uint32_t o[RD][4];
#pragma unroll
            for (int r = 0; r < RD; ++r)
                asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];"
                             : "=r"(o[r][0]), "=r"(o[r][1]), "=r"(o[r][2]), "=r"(o[r][3])
                             : "r"(otab + r * (CH * OW) + cg * 16)
                             : "memory");
#pragma unroll
            for (int r = 0; r < RD; ++r) {
                if constexpr (OW == 2) {
#pragma unroll
                    for (int h = 0; h < 4; ++h) {
                        const uint32_t a0 = (o[r][h] & 0xffffu) * four + rows;
                        const uint32_t a1 = (o[r][h] >> 16) * four + rows;
                        RowPair<MODE, VW, RJ, FM>::run(acc[r], a0, a1, one, cg == 0 && h == 0);
                    }
                } else {
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        const uint32_t a0 = o[r][2 * h] * one + rows;
                        const uint32_t a1 = o[r][2 * h + 1] * one + rows;
                        RowPair<MODE, VW, RJ, FM>::run(acc[r], a0, a1, one, cg == 0 && h == 0);
                    }
                }
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_empty + 8u * s);
        if constexpr (MODE == DD_U4) {  // the stage's byte lanes -> 16-bit lanes
#pragma unroll
            for (int r = 0; r < RD; ++r)
#pragma unroll
                for (int i = 0; i < RJ; ++i)
#pragma unroll
                    for (int v = 0; v < VW; ++v) acc[r][i][v].flush();
        }
        // the packed 16-bit lanes hold at most FLUSH_CH channels between flushes
        since_flush += CH;
        if (Acc<MODE, FM>::kNeedsFlush && since_flush + CH > FLUSH_CH) {
            since_flush = 0;
            if constexpr (TMEM) {
                if (k + 1 < p.nk) {  // (the last stage's sums go straight to the epilogue)
                    const uint32_t taddr = tmem_addr();
#pragma unroll
                    for (int ch = 0; ch < NCOL / 16; ++ch) {
                        uint32_t t[16];
                        if (parked) {
                            tmem_ld16(taddr + ch * 16, t);
                        } else {
#pragma unroll
                            for (int q = 0; q < 16; ++q) t[q] = 0u;
                        }
#pragma unroll
                        for (int q = 0; q < WPC; ++q) {
                            const int wi = ch * WPC + q;
                            uint32_t val[LPW];
                            acc[wi / (RJ * VW)][(wi / VW) % RJ][wi % VW].drain(val);
#pragma unroll
                            for (int l = 0; l < LPW; ++l) t[q * LPW + l] += val[l];
                        }
                        tmem_st16(taddr + ch * 16, t);
                    }
                    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
                    parked = true;
                }
            } else {
#pragma unroll
                for (int r = 0; r < RD; ++r)
#pragma unroll
                    for (int i = 0; i < RJ; ++i)
#pragma unroll
                        for (int v = 0; v < VW; ++v) acc[r][i][v].flush();
            }
        }
        if (++s == nstage) {
            s = 0;
            phase ^= 1u;
        }
    }

    // ========================= store (a7): lane l of superword j is output sample l*L + j
    // (the CTA's tile is recomputed here instead of being kept in registers across the hot loop)
    int b, jt;
    {
        int bid = blockIdx.x;
        asm volatile("" : "+r"(bid));
        tile_of_cta(p, bid, b, jt);
    }
    const int64_t j0 = static_cast<int64_t>(jt) * D_J;
    if constexpr (TMEM) {
        const uint32_t taddr = tmem_addr();
#pragma unroll
        for (int ch = 0; ch < NCOL / 16; ++ch) {
            uint32_t t[16];
            if (parked) {
                tmem_ld16(taddr + ch * 16, t);
            } else {
#pragma unroll
                for (int q = 0; q < 16; ++q) t[q] = 0u;
            }
#pragma unroll
            for (int q = 0; q < WPC; ++q) {
                const int wi = ch * WPC + q;
                const int r = wi / (RJ * VW), i = (wi / VW) % RJ, v = wi % VW;
                uint32_t val[LPW];
                acc[r][i][v].drain(val);
                const int d = b * D_DM + wd * RD + r;
                const int64_t j = j0 + (wj * RJ + i) * 32 + lane;
                if (d < p.ndm && j < p.L) {
                    uint32_t *o = static_cast<uint32_t *>(p.out) + static_cast<size_t>(d) * p.out_pitch;
#pragma unroll
                    for (int l = 0; l < LPW; ++l) {
                        const int64_t tt = static_cast<int64_t>(v * LPW + l) * p.L + j;
                        if (tt < p.out_len) o[tt] = t[q * LPW + l] + val[l];
                    }
                }
            }
        }
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        asm volatile("bar.sync 1, %0;" ::"r"((NCW + 1) * 32) : "memory");
        if (warp == 0) {
            uint32_t tmem;
            asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem) : "r"(bar_full + 960u) : "memory");
            asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(TCOLS) : "memory");
        }
        return;
    }
#pragma unroll
    for (int r = 0; r < RD; ++r) {
        const int d = b * D_DM + wd * RD + r;
        if (d >= p.ndm) continue;
#pragma unroll
        for (int i = 0; i < RJ; ++i) {
            const int64_t j = j0 + (wj * RJ + i) * 32 + lane;
            if (j >= p.L) continue;
#pragma unroll
            for (int v = 0; v < VW; ++v) {
                uint32_t val[LPW] = {};
                if constexpr (MODE == DD_U8) {
                    Acc<DD_U8, FM> &a = acc[r][i][v];
                    a.flush();
                    val[0] = a.a0;
                    val[1] = a.a1;
                    val[2] = a.a2;
                    val[3] = a.a3;
                } else if constexpr (MODE == DD_U16) {
                    Acc<DD_U16, FM> &a = acc[r][i][v];
                    val[0] = a.W - (a.H << 16);
                    val[1] = a.H;
                } else if constexpr (MODE == DD_F32) {
                    val[0] = __float_as_uint(acc[r][i][v].s);
                }
                uint32_t *o = static_cast<uint32_t *>(p.out) + static_cast<size_t>(d) * p.out_pitch;
#pragma unroll
                for (int l = 0; l < LPW; ++l) {
                    const int64_t t = static_cast<int64_t>(v * LPW + l) * p.L + j;
                    if (t < p.out_len) o[t] = val[l];
                }
            }
        }
    }
}

// ------------------------------------------------------------------ interleave pre-pass
// One thread makes four consecutive superwords (16*VW bytes, VW 16-byte stores) of one
// channel from LANES four-sample segments of the input row.  Reads past the end of a row
// (t >= nsamps) give 0; such lanes only feed outputs that are never stored.
template <typename T>
__device__ __forceinline__ uint32_t sample_or_zero(const T *row, int64_t t, int64_t nsamps)
{
    return t < nsamps ? static_cast<uint32_t>(row[t]) : 0u;
}

template <int MODE, int VW>
__global__ void __launch_bounds__(256) interleave_kernel(const InterleaveParams p)
{
    const int c = static_cast<int>(blockIdx.x / p.nchunk);
    const int64_t j = p.j_begin + (static_cast<int64_t>(blockIdx.x % p.nchunk) * blockDim.x + threadIdx.x) * 4;
    if (j >= p.j_end) return;
    uint32_t w[4 * VW];  // w[q * VW + v] = word v of superword j + q
    if (c >= p.nchans) {  // padding channel (nchans rounded up to CH): a zero row
#pragma unroll
        for (int i = 0; i < 4 * VW; ++i) w[i] = 0u;
    } else if (MODE == DD_U8) {
        const uint8_t *row = static_cast<const uint8_t *>(p.in) + static_cast<size_t>(c) * p.in_pitch;
        const bool aligned = (reinterpret_cast<uintptr_t>(row) & 3u) == 0;
        // every lane segment in range: issue all 4*VW loads before any is used
        const bool fast = aligned && (4 * VW - 1) * p.L + j + 3 < p.nsamps;
        uint32_t pre[VW][4];
        if (fast) {
#pragma unroll
            for (int v = 0; v < VW; ++v)
#pragma unroll
                for (int k = 0; k < 4; ++k)
                    pre[v][k] = *reinterpret_cast<const uint32_t *>(row + (v * 4 + k) * p.L + j);
        }
#pragma unroll
        for (int v = 0; v < VW; ++v) {
            uint32_t seg[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const int64_t t = (v * 4 + k) * p.L + j;
                if (fast) {
                    seg[k] = pre[v][k];
                } else if (aligned && t + 3 < p.nsamps) {
                    seg[k] = *reinterpret_cast<const uint32_t *>(row + t);
                } else {
                    seg[k] = sample_or_zero(row, t, p.nsamps) | sample_or_zero(row, t + 1, p.nsamps) << 8 |
                             sample_or_zero(row, t + 2, p.nsamps) << 16 |
                             sample_or_zero(row, t + 3, p.nsamps) << 24;
                }
            }
            // 4x4 byte transpose: word q gets byte q of each segment
            const uint32_t t01l = __byte_perm(seg[0], seg[1], 0x5140);  // a0 b0 a1 b1
            const uint32_t t01h = __byte_perm(seg[0], seg[1], 0x7362);  // a2 b2 a3 b3
            const uint32_t t23l = __byte_perm(seg[2], seg[3], 0x5140);
            const uint32_t t23h = __byte_perm(seg[2], seg[3], 0x7362);
            w[0 * VW + v] = __byte_perm(t01l, t23l, 0x5410);
            w[1 * VW + v] = __byte_perm(t01l, t23l, 0x7632);
            w[2 * VW + v] = __byte_perm(t01h, t23h, 0x5410);
            w[3 * VW + v] = __byte_perm(t01h, t23h, 0x7632);
        }
    } else if (MODE == DD_U16) {
        const uint16_t *row = static_cast<const uint16_t *>(p.in) + static_cast<size_t>(c) * p.in_pitch;
        const bool aligned = (reinterpret_cast<uintptr_t>(row) & 7u) == 0;
        const bool fast = aligned && (2 * VW - 1) * p.L + j + 3 < p.nsamps;  // all loads up front
        uint2 pre[VW][2];
        if (fast) {
#pragma unroll
            for (int v = 0; v < VW; ++v)
#pragma unroll
                for (int k = 0; k < 2; ++k)
                    pre[v][k] = *reinterpret_cast<const uint2 *>(row + (v * 2 + k) * p.L + j);
        }
#pragma unroll
        for (int v = 0; v < VW; ++v) {
            uint2 seg[2];
#pragma unroll
            for (int k = 0; k < 2; ++k) {
                const int64_t t = (v * 2 + k) * p.L + j;
                if (fast) {
                    seg[k] = pre[v][k];
                } else if (aligned && t + 3 < p.nsamps) {
                    seg[k] = *reinterpret_cast<const uint2 *>(row + t);
                } else {
                    seg[k].x = sample_or_zero(row, t, p.nsamps) | sample_or_zero(row, t + 1, p.nsamps) << 16;
                    seg[k].y = sample_or_zero(row, t + 2, p.nsamps) | sample_or_zero(row, t + 3, p.nsamps) << 16;
                }
            }
            w[0 * VW + v] = __byte_perm(seg[0].x, seg[1].x, 0x5410);
            w[1 * VW + v] = __byte_perm(seg[0].x, seg[1].x, 0x7632);
            w[2 * VW + v] = __byte_perm(seg[0].y, seg[1].y, 0x5410);
            w[3 * VW + v] = __byte_perm(seg[0].y, seg[1].y, 0x7632);
        }
    } else {
        const uint32_t *row = static_cast<const uint32_t *>(p.in) + static_cast<size_t>(c) * p.in_pitch;
        const bool aligned = (reinterpret_cast<uintptr_t>(row) & 15u) == 0;
        const bool fast = aligned && (VW - 1) * p.L + j + 3 < p.nsamps;  // all loads up front
        uint4 pre[VW];
        if (fast) {
#pragma unroll
            for (int v = 0; v < VW; ++v) pre[v] = *reinterpret_cast<const uint4 *>(row + v * p.L + j);
        }
#pragma unroll
        for (int v = 0; v < VW; ++v) {
            const int64_t t = v * p.L + j;
            uint4 seg;
            if (fast) {
                seg = pre[v];
            } else if (aligned && t + 3 < p.nsamps) {
                seg = *reinterpret_cast<const uint4 *>(row + t);
            } else {
                seg.x = sample_or_zero(row, t, p.nsamps);
                seg.y = sample_or_zero(row, t + 1, p.nsamps);
                seg.z = sample_or_zero(row, t + 2, p.nsamps);
                seg.w = sample_or_zero(row, t + 3, p.nsamps);
            }
            w[0 * VW + v] = seg.x;
            w[1 * VW + v] = seg.y;
            w[2 * VW + v] = seg.z;
            w[3 * VW + v] = seg.w;
        }
    }
    uint4 *dst = reinterpret_cast<uint4 *>(p.X + (static_cast<size_t>(c) * p.Lw + j) * VW);
#pragma unroll
    for (int i = 0; i < VW; ++i) dst[i] = make_uint4(w[4 * i], w[4 * i + 1], w[4 * i + 2], w[4 * i + 3]);
}

// 8 x 8 transpose of 4-bit elements: on entry nibble q of r[n] is element (n, q), on return
// nibble n of r[q] is element (n, q).  16-bit and 8-bit block swaps with PRMT, the last level
// with shifts and masks (32 instructions for 64 elements).
__device__ __forceinline__ void transpose_nibbles_8x8(uint32_t (&r)[8])
{
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const uint32_t a = r[i], b = r[i + 4];
        r[i] = __byte_perm(a, b, 0x5410);
        r[i + 4] = __byte_perm(a, b, 0x7632);
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        if (i & 2) continue;
        const uint32_t a = r[i], b = r[i + 2];
        r[i] = __byte_perm(a, b, 0x6240);
        r[i + 2] = __byte_perm(a, b, 0x7351);
    }
#pragma unroll
    for (int i = 0; i < 8; i += 2) {
        const uint32_t a = r[i], b = r[i + 1];
        r[i] = (a & 0x0F0F0F0Fu) | ((b << 4) & 0xF0F0F0F0u);
        r[i + 1] = ((a >> 4) & 0x0F0F0F0Fu) | (b & 0xF0F0F0F0u);
    }
}

// Packed 4-bit rows (two samples per byte, the earlier one in the low nibble; DESIGN.md reading
// R14) -> superwords of VW words of EIGHT 4-bit lanes: nibble n of word v of X[c][j] is
// in[c][(8v + n)*L + j].  One thread makes eight consecutive superwords of one channel from
// 8*VW eight-sample segments (one 32-bit load each) and VW 8 x 8 nibble transposes.
template <int VW>
__global__ void __launch_bounds__(256) interleave_u4_kernel(const InterleaveParams p)
{
    const int c = static_cast<int>(blockIdx.x / p.nchunk);
    const int64_t j = p.j_begin + (static_cast<int64_t>(blockIdx.x % p.nchunk) * blockDim.x + threadIdx.x) * 8;
    if (j >= p.j_end) return;
    uint32_t w[VW][8];  // w[v][q] = word v of superword j + q
    if (c >= p.nchans) {
#pragma unroll
        for (int v = 0; v < VW; ++v)
#pragma unroll
            for (int q = 0; q < 8; ++q) w[v][q] = 0u;
    } else {
        const uint8_t *row = static_cast<const uint8_t *>(p.in) + static_cast<size_t>(c) * (p.in_pitch / 2);
        const bool aligned = (reinterpret_cast<uintptr_t>(row) & 3u) == 0;
        // every segment in range: issue all loads before any is used
        const bool fast = aligned && (8 * VW - 1) * p.L + j + 7 < p.nsamps;
        if (fast) {
#pragma unroll
            for (int v = 0; v < VW; ++v)
#pragma unroll
                for (int n = 0; n < 8; ++n)
                    w[v][n] = *reinterpret_cast<const uint32_t *>(row + (((v * 8 + n) * p.L + j) >> 1));
        } else {
#pragma unroll
            for (int v = 0; v < VW; ++v)
#pragma unroll
                for (int n = 0; n < 8; ++n) {
                    const int64_t t = (v * 8 + n) * p.L + j;  // multiple of 8: starts on a byte
                    uint32_t x = 0u;
                    if (aligned && t + 7 < p.nsamps) {
                        x = *reinterpret_cast<const uint32_t *>(row + (t >> 1));
                    } else {
#pragma unroll
                        for (int k = 0; k < 4; ++k) {
                            uint32_t byte = 0u;
                            if (t + 2 * k < p.nsamps) byte = row[(t >> 1) + k];
                            if (t + 2 * k + 1 >= p.nsamps) byte &= 0x0Fu;  // odd valid length: drop the nibble past the end
                            x |= byte << (8 * k);
                        }
                    }
                    w[v][n] = x;
                }
        }
#pragma unroll
        for (int v = 0; v < VW; ++v) transpose_nibbles_8x8(w[v]);
    }
    uint32_t *dst = p.X + (static_cast<size_t>(c) * p.Lw + j) * VW;
    if constexpr (VW == 1) {
        *reinterpret_cast<uint4 *>(dst) = make_uint4(w[0][0], w[0][1], w[0][2], w[0][3]);
        *reinterpret_cast<uint4 *>(dst + 4) = make_uint4(w[0][4], w[0][5], w[0][6], w[0][7]);
    } else if constexpr (VW == 2) {
#pragma unroll
        for (int q = 0; q < 8; q += 2)
            *reinterpret_cast<uint4 *>(dst + q * 2) = make_uint4(w[0][q], w[1][q], w[0][q + 1], w[1][q + 1]);
    } else {
#pragma unroll
        for (int q = 0; q < 8; ++q)
            *reinterpret_cast<uint4 *>(dst + q * 4) = make_uint4(w[0][q], w[1][q], w[2][q], w[3][q]);
    }
}

// ------------------------------------------------------------------ transpose pre-step
// Time-major filterbank [nsamps][nchans] (how telescopes write it) -> channel-major
// [nchans][nsamps] (what Eq. 3 / Alg. 3 index); the paper counts this step
// in its pipeline time.  HBM-bound: every byte is read once and written once.
// A CTA moves a tile of TC = 32*P channels x 128 samples (P = elements per 32-bit word; 16 KB).
// Phase 1: a thread loads P words from P consecutive time rows (coalesced along channels),
// sixteen words in flight, transposes the P x P elements in registers and stores P words into
// the transposed shared-memory tile.  Phase 2: rows of that tile (one channel, 128 samples) go
// out as coalesced word stores; an output row that does not start on a 4-byte boundary
// (nsamps not a multiple of 4 bytes) gets its words funnel-shifted into place, the few head and
// tail bytes stored one by one.  Ragged edge tiles and time rows that are not 4-byte aligned
// take an element-wise path through the same tile.
template <typename T>
__global__ void __launch_bounds__(256) transpose_kernel(const TransposeParams p)
{
    constexpr int E = static_cast<int>(sizeof(T));
    constexpr int P = 4 / E;
    constexpr int TC = 32 * P, TT = 128;
    constexpr int WT = TT / P;  // words per tile row
    // [channel row][word along time], +1 word of pitch; channel c of the tile lives in row
    // phys(c) = (c % P) * 32 + c / P so that the 32 lanes of a phase-1 store (consecutive channel
    // words, same k = c % P) hit 32 different banks
    __shared__ uint32_t tile[TC][WT + 1];
    auto phys = [](int c) { return (c % P) * 32 + c / P; };
    const T *in = static_cast<const T *>(p.in);
    T *out = static_cast<T *>(p.out);
    const int64_t t0 = static_cast<int64_t>(blockIdx.x) * TT;
    const int c0 = static_cast<int>(blockIdx.y) * TC;
    const bool full = t0 + TT <= p.nsamps && c0 + TC <= p.nchans;
    const bool in_al = (reinterpret_cast<uintptr_t>(in) & 3u) == 0 && (p.nchans * E) % 4 == 0;
    const bool out_ok = (reinterpret_cast<uintptr_t>(out) & (E - 1)) == 0;
    if (full && in_al && out_ok) {
        constexpr int NU = TT / P / 8;  // groups of P time rows per thread
        uint32_t rr[NU][P];             // all 16 loads of the thread in flight before any is used
#pragma unroll
        for (int u = 0; u < NU; ++u) {
            const int q = threadIdx.x + 256 * u;
            const int cg = q & 31, tg = q >> 5;
#pragma unroll
            for (int i = 0; i < P; ++i)
                rr[u][i] = *reinterpret_cast<const uint32_t *>(in + (t0 + tg * P + i) * p.nchans + c0 + cg * P);
        }
#pragma unroll
        for (int u = 0; u < NU; ++u) {
            const int q = threadIdx.x + 256 * u;
            const int cg = q & 31, tg = q >> 5;  // word along channels, group of P time rows
            uint32_t r[P];
#pragma unroll
            for (int i = 0; i < P; ++i) r[i] = rr[u][i];
            if constexpr (P == 4) {
                const uint32_t a = __byte_perm(r[0], r[1], 0x5140), b = __byte_perm(r[0], r[1], 0x7362);
                const uint32_t c = __byte_perm(r[2], r[3], 0x5140), d = __byte_perm(r[2], r[3], 0x7362);
                tile[0 * 32 + cg][tg] = __byte_perm(a, c, 0x5410);
                tile[1 * 32 + cg][tg] = __byte_perm(a, c, 0x7632);
                tile[2 * 32 + cg][tg] = __byte_perm(b, d, 0x5410);
                tile[3 * 32 + cg][tg] = __byte_perm(b, d, 0x7632);
            } else if constexpr (P == 2) {
                tile[0 * 32 + cg][tg] = __byte_perm(r[0], r[1], 0x5410);
                tile[1 * 32 + cg][tg] = __byte_perm(r[0], r[1], 0x7632);
            } else {
                tile[cg][tg] = r[0];
            }
        }
        __syncthreads();
        // a warp writes one tile row (or WT / 32 warps share one) per step
        const int64_t pitch_b = p.nsamps * E;
        unsigned char *tile_out = reinterpret_cast<unsigned char *>(out + static_cast<int64_t>(c0) * p.nsamps + t0);
#pragma unroll 4
        for (int q = threadIdx.x; q < TC * WT; q += 256) {
            const int w = q % WT, r = q / WT;
            const int c = (r % 32) * P + r / 32;  // inverse of phys
            unsigned char *row = tile_out + c * pitch_b;
            const uint32_t e = (0u - static_cast<uint32_t>(reinterpret_cast<uintptr_t>(row))) & 3u;  // head bytes
            const uint32_t lo = tile[r][w];
            if (e == 0) {
                reinterpret_cast<uint32_t *>(row)[w] = lo;
            } else {
                if (w < WT - 1) *reinterpret_cast<uint32_t *>(row + e + 4 * w) = __funnelshift_r(lo, tile[r][w + 1], 8 * e);
                // the row's e head bytes and 4 - e tail bytes: byte i of the first / last word
                if (w < 4) {
                    const bool head = static_cast<uint32_t>(w) < e;
                    const uint32_t word = tile[r][head ? 0 : WT - 1];
                    row[head ? w : 4 * (WT - 1) + w] = static_cast<unsigned char>(word >> (8 * w));
                }
            }
        }
        return;
    }
    T *te = reinterpret_cast<T *>(&tile[0][0]);  // element view: row pitch WT + 1 words
    for (int q = threadIdx.x; q < TC * TT; q += 256) {
        const int c = q % TC, t = q / TC;
        T v = 0;
        if (t0 + t < p.nsamps && c0 + c < p.nchans) v = in[(t0 + t) * p.nchans + c0 + c];
        te[phys(c) * ((WT + 1) * P) + t] = v;
    }
    __syncthreads();
    for (int q = threadIdx.x; q < TC * TT; q += 256) {
        const int t = q % TT, c = q / TT;
        if (t0 + t < p.nsamps && c0 + c < p.nchans)
            out[static_cast<int64_t>(c0 + c) * p.nsamps + t0 + t] = te[phys(c) * ((WT + 1) * P) + t];
    }
}

// Packed 4-bit: time-major [nsamps][nchans/2 bytes] (even channel of a byte in the low nibble,
// reading R16) -> channel-major [nchans][nsamps/2 bytes] (earlier sample in the low nibble, R14).
// A CTA moves 256 channels x 256 samples.  Two time rows are first merged nibble-wise into the
// bytes of the even channels and of the odd channels ((t, t+1) of one channel = one output byte);
// what is left is the byte transpose of transpose_kernel<uint8_t>, once per channel parity.
__global__ void __launch_bounds__(256) transpose_u4_kernel(const TransposeParams p)
{
    constexpr int TC = 256, TU = 128;  // channels, output bytes (pairs of samples) per tile
    constexpr int WT = TU / 4;         // words per tile row
    __shared__ uint32_t tile[TC][WT + 1];  // row phys(c) = (c % 8) * 32 + c / 8
    const uint8_t *in = static_cast<const uint8_t *>(p.in);
    uint8_t *out = static_cast<uint8_t *>(p.out);
    const int64_t in_pitch = p.nchans / 2, out_pitch = p.nsamps / 2;  // bytes per input / output row
    const int64_t u0 = static_cast<int64_t>(blockIdx.x) * TU;         // first output byte column
    const int c0 = static_cast<int>(blockIdx.y) * TC;
    const bool full = 2 * (u0 + TU) <= p.nsamps && c0 + TC <= p.nchans;
    const bool in_al = (reinterpret_cast<uintptr_t>(in) & 3u) == 0 && in_pitch % 4 == 0;
    if (full && in_al) {
#pragma unroll
        for (int half = 0; half < 2; ++half) {  // 2 x 2 groups of (word of 8 channels) x (4 output bytes)
            uint32_t rr[2][8];
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                const int q = threadIdx.x + 256 * (2 * half + u);
                const int cg = q & 31, ug = q >> 5;
#pragma unroll
                for (int i = 0; i < 8; ++i)
                    rr[u][i] = *reinterpret_cast<const uint32_t *>(in + (2 * u0 + 8 * ug + i) * in_pitch + c0 / 2 + cg * 4);
            }
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                const int q = threadIdx.x + 256 * (2 * half + u);
                const int cg = q & 31, ug = q >> 5;
                uint32_t ev[4], od[4];
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    const uint32_t a = rr[u][2 * i], b = rr[u][2 * i + 1];  // samples 2k and 2k+1 of 8 channels
                    ev[i] = (a & 0x0F0F0F0Fu) | ((b & 0x0F0F0F0Fu) << 4);
                    od[i] = ((a >> 4) & 0x0F0F0F0Fu) | (b & 0xF0F0F0F0u);
                }
#pragma unroll
                for (int par = 0; par < 2; ++par) {
                    const uint32_t *x = par ? od : ev;  // byte j of x[i]: channel 8 cg + 2 j + par, output byte 4 ug + i
                    const uint32_t a = __byte_perm(x[0], x[1], 0x5140), b = __byte_perm(x[0], x[1], 0x7362);
                    const uint32_t c = __byte_perm(x[2], x[3], 0x5140), d = __byte_perm(x[2], x[3], 0x7362);
                    tile[(0 + par) * 32 + cg][ug] = __byte_perm(a, c, 0x5410);
                    tile[(2 + par) * 32 + cg][ug] = __byte_perm(a, c, 0x7632);
                    tile[(4 + par) * 32 + cg][ug] = __byte_perm(b, d, 0x5410);
                    tile[(6 + par) * 32 + cg][ug] = __byte_perm(b, d, 0x7632);
                }
            }
        }
        __syncthreads();
        unsigned char *tile_out = out + static_cast<int64_t>(c0) * out_pitch + u0;
#pragma unroll 4
        for (int q = threadIdx.x; q < TC * WT; q += 256) {
            const int w = q % WT, r = q / WT;
            const int c = (r % 32) * 8 + r / 32;  // inverse of phys
            unsigned char *row = tile_out + c * out_pitch;
            const uint32_t e = (0u - static_cast<uint32_t>(reinterpret_cast<uintptr_t>(row))) & 3u;  // head bytes
            const uint32_t lo = tile[r][w];
            if (e == 0) {
                reinterpret_cast<uint32_t *>(row)[w] = lo;
            } else {
                if (w < WT - 1) *reinterpret_cast<uint32_t *>(row + e + 4 * w) = __funnelshift_r(lo, tile[r][w + 1], 8 * e);
                if (w < 4) {
                    const bool head = static_cast<uint32_t>(w) < e;
                    const uint32_t word = tile[r][head ? 0 : WT - 1];
                    row[head ? w : 4 * (WT - 1) + w] = static_cast<unsigned char>(word >> (8 * w));
                }
            }
        }
        return;
    }
    // ragged tiles and unaligned time rows: one output byte per step
    for (int q = threadIdx.x; q < TC * TU; q += 256) {
        const int u = q % TU, c = q / TU;
        const int64_t t = 2 * (u0 + u);
        if (t >= p.nsamps || c0 + c >= p.nchans) continue;
        const int sh = ((c0 + c) & 1) * 4;
        const uint32_t a = in[t * in_pitch + (c0 + c) / 2] >> sh, b = in[(t + 1) * in_pitch + (c0 + c) / 2] >> sh;
        out[static_cast<int64_t>(c0 + c) * out_pitch + u0 + u] = static_cast<uint8_t>((a & 15u) | (b & 15u) << 4);
    }
}

// ------------------------------------------------------------------ fused transpose + interleave
// Time-major input [nsamps][nchans] straight into the lane-interleaved workspace X (what
// transpose_kernel + interleave_kernel do in two HBM round trips).  A CTA owns TC = 128 bytes
// of channels x 32 superword columns.  Phase 1: for each of the LANES x 32 time rows the tile
// needs (t = l*L + j), one warp copies the row's 128 bytes (word loads, coalesced along
// channels) into shared memory.  Phase 2: a thread gathers the LANES elements of one
// (channel, column) superword (byte/half/word loads at a 33-word row pitch: conflict-free
// across the 32 columns of a warp) and stores it; a warp writes 32 consecutive superwords.
template <typename T, int VW>
__global__ void __launch_bounds__(256) interleave_tm_kernel(const InterleaveParams p)
{
    constexpr int E = static_cast<int>(sizeof(T));
    constexpr int LPW = 4 / E, NL = VW * LPW;
    constexpr int TC = 128 / E;               // channels per tile
    constexpr int TJ = NL > 8 ? 16 : 32;      // superword columns per tile (static smem <= 48 KB)
    __shared__ uint32_t tile[NL * TJ][33];
    const T *in = static_cast<const T *>(p.in);
    const int64_t ncol_tiles = (p.Lw + TJ - 1) / TJ;
    const int64_t j0 = static_cast<int64_t>(blockIdx.x % ncol_tiles) * TJ;
    const int c0 = static_cast<int>(blockIdx.x / ncol_tiles) * TC;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const bool in_al = (reinterpret_cast<uintptr_t>(in) & 3u) == 0 && (p.in_pitch * E) % 4 == 0;
    // ---- phase 1: rows r = l*TJ + j  <->  time l*L + j0 + j, channels c0 .. c0+TC
    const bool fast = in_al && c0 + TC <= p.nchans;
    if (fast) {  // all loads of a warp first (NL*TJ/8 independent 128-byte rows in flight), then the stores
        constexpr int NR = NL * TJ / 8;
        uint32_t w[NR];
#pragma unroll
        for (int i = 0; i < NR; ++i) {
            const int r = warp + 8 * i;
            const int64_t t = static_cast<int64_t>(r / TJ) * p.L + j0 + (r % TJ);
            w[i] = t < p.nsamps ? reinterpret_cast<const uint32_t *>(in + t * p.in_pitch + c0)[lane] : 0u;
        }
#pragma unroll
        for (int i = 0; i < NR; ++i) tile[warp + 8 * i][lane] = w[i];
    }
    for (int r = warp; !fast && r < NL * TJ; r += 8) {
        const int64_t t = static_cast<int64_t>(r / TJ) * p.L + j0 + (r % TJ);
        uint32_t w = 0u;
        if (t < p.nsamps) {
            const T *src = in + t * p.in_pitch + c0;  // in_pitch = nchans: elements per time row
#pragma unroll
            for (int k = 0; k < LPW; ++k) {
                const int c = c0 + lane * LPW + k;
                if (c < p.nchans) w |= static_cast<uint32_t>(src[lane * LPW + k]) << (8 * E * k);
            }
        }
        tile[r][lane] = w;
    }
    __syncthreads();
    // ---- phase 2: a thread takes one column j and one 32-bit word column cw (LPW channels):
    // it loads that word from each of the NL lane rows (row pitch 33 words: conflict-free
    // across the columns of a warp), transposes LPW x LPW elements per superword word in
    // registers and stores LPW superwords (channels cw*LPW + k), each store coalesced along j
    for (int q = threadIdx.x; q < 32 * TJ; q += 256) {
        const int j = q % TJ, cw = q / TJ;
        if (j0 + j >= p.Lw) continue;
        uint32_t wl[NL];
#pragma unroll
        for (int l = 0; l < NL; ++l) wl[l] = tile[l * TJ + j][cw];
        uint32_t o[LPW][VW];  // o[k][v]: word v of channel cw*LPW + k
#pragma unroll
        for (int v = 0; v < VW; ++v) {
            if constexpr (LPW == 4) {
                const uint32_t a = __byte_perm(wl[4 * v], wl[4 * v + 1], 0x5140), b2 = __byte_perm(wl[4 * v], wl[4 * v + 1], 0x7362);
                const uint32_t c2 = __byte_perm(wl[4 * v + 2], wl[4 * v + 3], 0x5140), d2 = __byte_perm(wl[4 * v + 2], wl[4 * v + 3], 0x7362);
                o[0][v] = __byte_perm(a, c2, 0x5410);
                o[1][v] = __byte_perm(a, c2, 0x7632);
                o[2][v] = __byte_perm(b2, d2, 0x5410);
                o[3][v] = __byte_perm(b2, d2, 0x7632);
            } else if constexpr (LPW == 2) {
                o[0][v] = __byte_perm(wl[2 * v], wl[2 * v + 1], 0x5410);
                o[1][v] = __byte_perm(wl[2 * v], wl[2 * v + 1], 0x7632);
            } else {
                o[0][v] = wl[v];
            }
        }
#pragma unroll
        for (int k = 0; k < LPW; ++k) {
            const int c = c0 + cw * LPW + k;
            if (c >= p.nrows) continue;
            uint32_t *dst = p.X + (static_cast<size_t>(c) * p.Lw + j0 + j) * VW;
            if constexpr (VW == 1)
                dst[0] = o[k][0];
            else if constexpr (VW == 2)
                *reinterpret_cast<uint2 *>(dst) = make_uint2(o[k][0], o[k][1]);
            else
                *reinterpret_cast<uint4 *>(dst) = make_uint4(o[k][0], o[k][1], o[k][2], o[k][3]);
        }
    }
}

// The same for packed 4-bit time-major input [nsamps][nchans/2 bytes] (reading R16: the even
// channel of a byte in the low nibble), into the eight-lanes-per-word layout of
// interleave_u4_kernel: a tile is 128 bytes = 256 channels x TJ superword columns; in phase 2 a
// thread takes the words of one column and eight channels from the 8*VW lane rows, transposes
// 8 x 8 nibbles per superword word (lane <-> channel) and stores the superwords of its channels.
template <int VW>
__global__ void __launch_bounds__(256) interleave_tm_u4_kernel(const InterleaveParams p)
{
    constexpr int NL = VW * 8;
    constexpr int TJ = 256 / NL;
    __shared__ uint32_t tile[NL * TJ][33];
    const uint8_t *in = static_cast<const uint8_t *>(p.in);
    const int64_t pb = p.in_pitch / 2;  // bytes per time row
    const int64_t ncol_tiles = (p.Lw + TJ - 1) / TJ;
    const int64_t j0 = static_cast<int64_t>(blockIdx.x % ncol_tiles) * TJ;
    const int c0 = static_cast<int>(blockIdx.x / ncol_tiles) * 256;  // first channel of the tile
    const int b0 = c0 / 2;                                           // its byte in a time row
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const bool fast = (reinterpret_cast<uintptr_t>(in) & 3u) == 0 && pb % 4 == 0 && b0 + 128 <= pb;
    constexpr int NR = NL * TJ / 8;
    if (fast) {
        uint32_t w[NR];
#pragma unroll
        for (int i = 0; i < NR; ++i) {
            const int r = warp + 8 * i;
            const int64_t t = static_cast<int64_t>(r / TJ) * p.L + j0 + (r % TJ);
            w[i] = t < p.nsamps ? reinterpret_cast<const uint32_t *>(in + t * pb + b0)[lane] : 0u;
        }
#pragma unroll
        for (int i = 0; i < NR; ++i) tile[warp + 8 * i][lane] = w[i];
    } else {
        for (int r = warp; r < NL * TJ; r += 8) {
            const int64_t t = static_cast<int64_t>(r / TJ) * p.L + j0 + (r % TJ);
            uint32_t w = 0u;
            if (t < p.nsamps) {
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const int64_t b = b0 + lane * 4 + k;
                    if (b < pb) w |= static_cast<uint32_t>(in[t * pb + b]) << (8 * k);
                }
            }
            tile[r][lane] = w;
        }
    }
    __syncthreads();
    for (int q = threadIdx.x; q < 32 * TJ; q += 256) {
        const int j = q % TJ, cw = q / TJ;
        if (j0 + j >= p.Lw) continue;
        uint32_t o[VW][8];  // o[v][k]: word v of channel c0 + cw*8 + k
#pragma unroll
        for (int v = 0; v < VW; ++v) {
#pragma unroll
            for (int n = 0; n < 8; ++n) o[v][n] = tile[(8 * v + n) * TJ + j][cw];  // nibble k = channel k at lane 8v + n
            transpose_nibbles_8x8(o[v]);
        }
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const int c = c0 + cw * 8 + k;
            if (c >= p.nrows) continue;
            uint32_t *dst = p.X + (static_cast<size_t>(c) * p.Lw + j0 + j) * VW;
            if constexpr (VW == 1)
                dst[0] = o[0][k];
            else if constexpr (VW == 2)
                *reinterpret_cast<uint2 *>(dst) = make_uint2(o[0][k], o[1][k]);
            else
                *reinterpret_cast<uint4 *>(dst) = make_uint4(o[0][k], o[1][k], o[2][k], o[3][k]);
        }
    }
}

// ------------------------------------------------------------------ time binning pre-step
// out[c][t] = sum_{i < F} in[c][F*t + i]  (PAPER.md:295, 370 name the step; reading R15 in
// raw sums, integer types widened -- u4 -> u8, u8 -> u16 -- float32 summed in
// ascending i).  HBM-bound: each input byte is read once.  A thread makes four consecutive
// outputs from 4*F consecutive inputs (word loads when the rows are 4-byte aligned).
template <int MODE>
__device__ __forceinline__ uint32_t bin_sample(const void *row, int64_t t)
{
    if (MODE == DD_U4) {
        const uint32_t b = static_cast<const uint8_t *>(row)[t >> 1];
        return (t & 1) ? b >> 4 : b & 15u;
    }
    return static_cast<const uint8_t *>(row)[t];
}

// Fast path for integer input whose rows are 16-byte aligned: one thread loads one 16-byte
// piece (16 u8 / 32 u4 samples = NO = 16/F or 32/F whole bins, F | 16), sums in registers and
// stores NO outputs with one vector store; four pieces per thread in flight.
template <int MODE, int F>
__global__ void __launch_bounds__(256) bin_time_fast_kernel(const BinParams p)
{
    constexpr int NS = MODE == DD_U4 ? 32 : 16;  // samples per piece
    constexpr int NO = NS / F;                   // outputs per piece
    constexpr int OB = MODE == DD_U4 ? 1 : 2;    // bytes per output
    const int64_t npiece = p.nout / NO;          // whole pieces per row (the rest: bin_time_kernel)
    const int64_t nchunk = (npiece + 1023) / 1024;
    const int c = static_cast<int>(blockIdx.x / nchunk);
    const size_t row_bytes = MODE == DD_U4 ? static_cast<size_t>(p.nsamps / 2) : static_cast<size_t>(p.nsamps);
    const uint4 *row = reinterpret_cast<const uint4 *>(static_cast<const uint8_t *>(p.in) + c * row_bytes);
    uint8_t *orow = static_cast<uint8_t *>(p.out) + static_cast<size_t>(c) * p.nout * OB;
    const int64_t q0 = static_cast<int64_t>(blockIdx.x % nchunk) * 1024 + threadIdx.x;
    uint4 v[4];
#pragma unroll
    for (int u = 0; u < 4; ++u)
        if (q0 + u * 256 < npiece) v[u] = row[q0 + u * 256];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
        const int64_t q = q0 + u * 256;
        if (q >= npiece) continue;
        const uint32_t w[4] = {v[u].x, v[u].y, v[u].z, v[u].w};
        uint32_t sum[NO];
#pragma unroll
        for (int o = 0; o < NO; ++o) sum[o] = 0u;
#pragma unroll
        for (int b = 0; b < 16; ++b) {
            const uint32_t byte = (w[b >> 2] >> (8 * (b & 3))) & 0xffu;
            if (MODE == DD_U4) {
                sum[(2 * b) / F] += byte & 15u;
                sum[(2 * b + 1) / F] += byte >> 4;
            } else {
                sum[b / F] += byte;
            }
        }
        uint32_t packed[(NO * OB + 3) / 4];
#pragma unroll
        for (int i = 0; i < (NO * OB + 3) / 4; ++i) packed[i] = 0u;
#pragma unroll
        for (int o = 0; o < NO; ++o) packed[(o * OB) >> 2] |= sum[o] << (8 * ((o * OB) & 3));
        uint8_t *dst = orow + q * (NO * OB);
        if constexpr (NO * OB == 16)
            *reinterpret_cast<uint4 *>(dst) = make_uint4(packed[0], packed[1], packed[2], packed[3]);
        else if constexpr (NO * OB == 8)
            *reinterpret_cast<uint2 *>(dst) = make_uint2(packed[0], packed[1]);
        else if constexpr (NO * OB == 4)
            *reinterpret_cast<uint32_t *>(dst) = packed[0];
        else if constexpr (NO * OB == 2)
            *reinterpret_cast<uint16_t *>(dst) = static_cast<uint16_t>(packed[0]);
        else
            *dst = static_cast<uint8_t>(packed[0]);
    }
}

// Integer input whose rows are NOT 16-byte aligned (e.g. 156250-sample rows): a piece is 16 bytes
// of OUTPUT (an aligned vector store; the first aligned output of a row depends on the row) made
// from 8*F input bytes, which start at any byte address: 2*F + 1 word loads from the 4-byte
// aligned address below it, funnel-shifted into place.  Sums are formed inside 32-bit words
// (pairs of bytes / nibbles, then dp4a).  The outputs of a row before its first and after its
// last whole piece -- and the row's last piece, whose funnel would read past the row -- are made
// one by one by one thread per row.  Needs in 4-byte aligned and out aligned to its element.
template <int MODE, int F>
__global__ void __launch_bounds__(256) bin_time_rows_kernel(const BinParams p)
{
    constexpr int OB = MODE == DD_U4 ? 1 : 2;  // bytes per output
    constexpr int NO = 16 / OB;                // outputs per piece
    constexpr int NW = 2 * F;                  // input words per piece (8*F bytes, both types)
    const int64_t nchunk = p.row_chunks;
    const int c = static_cast<int>(blockIdx.x / nchunk);
    const size_t row_bytes = MODE == DD_U4 ? static_cast<size_t>(p.nsamps / 2) : static_cast<size_t>(p.nsamps);
    const uint8_t *row = static_cast<const uint8_t *>(p.in) + c * row_bytes;
    uint8_t *orow = static_cast<uint8_t *>(p.out) + static_cast<size_t>(c) * p.nout * OB;
    int64_t head = static_cast<int64_t>((16u - (reinterpret_cast<uintptr_t>(orow) & 15u)) & 15u) / OB;
    if (head > p.nout) head = p.nout;
    int64_t npiece = (p.nout - head) / NO - 1;
    if (npiece < 0) npiece = 0;
    const int64_t q0 = static_cast<int64_t>(blockIdx.x % nchunk) * 512 + threadIdx.x;
    uint32_t w[2][NW + 1];
    const uint8_t *src[2];
#pragma unroll
    for (int u = 0; u < 2; ++u) {  // all loads of both pieces first
        const int64_t q = q0 + u * 256;
        if (q >= npiece) continue;
        const int64_t a = (head + q * NO) * F / (MODE == DD_U4 ? 2 : 1);  // first input byte of the piece
        src[u] = row + a;
        const uint32_t *al = reinterpret_cast<const uint32_t *>(reinterpret_cast<uintptr_t>(src[u]) & ~static_cast<uintptr_t>(3));
#pragma unroll
        for (int i = 0; i < NW; ++i) w[u][i] = al[i];
        w[u][NW] = (reinterpret_cast<uintptr_t>(src[u]) & 3u) ? al[NW] : 0u;
    }
#pragma unroll
    for (int u = 0; u < 2; ++u) {
        const int64_t q = q0 + u * 256;
        if (q >= npiece) continue;
        const uint32_t sh = static_cast<uint32_t>(reinterpret_cast<uintptr_t>(src[u]) & 3u) * 8u;
        uint32_t o[4];  // the 16 output bytes
        uint32_t part[NW];  // per input word: sums inside the word
#pragma unroll
        for (int i = 0; i < NW; ++i) {
            const uint32_t x = __funnelshift_r(w[u][i], w[u][i + 1], sh);
            if (MODE == DD_U4)
                part[i] = (x & 0x0F0F0F0Fu) + ((x >> 4) & 0x0F0F0F0Fu);  // 4 byte lanes: nibble pairs
            else
                part[i] = x;                                            // 4 byte lanes: samples
        }
        // byte lanes -> outputs.  G = byte lanes per output: u8 F, u4 F/2.
        constexpr int G = MODE == DD_U4 ? F / 2 : F;
        if constexpr (G == 1) {  // u4, F = 2: the byte lanes are the outputs (NW = 4 words = 16 outputs)
#pragma unroll
            for (int i = 0; i < 4; ++i) o[i] = part[i];
        } else if constexpr (G == 2) {  // two outputs per word as 16-bit lanes
            uint32_t h[NW];
#pragma unroll
            for (int i = 0; i < NW; ++i) h[i] = (part[i] & 0x00FF00FFu) + ((part[i] >> 8) & 0x00FF00FFu);
            if constexpr (OB == 2) {  // u8, F = 2: NW = 4 words of two u16 outputs
#pragma unroll
                for (int i = 0; i < 4; ++i) o[i] = h[i];
            } else {                  // u4, F = 4: NW = 8 words of two outputs -> bytes
#pragma unroll
                for (int i = 0; i < 4; ++i) o[i] = __byte_perm(h[2 * i], h[2 * i + 1], 0x6420);
            }
        } else {  // G >= 4: an output is the sum of G / 4 whole words' byte lanes (dp4a)
            constexpr int WPO = G / 4;
            uint32_t v[NO];
#pragma unroll
            for (int k = 0; k < NO; ++k) {
                uint32_t acc = 0u;
#pragma unroll
                for (int i = 0; i < WPO; ++i) acc = __dp4a(part[k * WPO + i], 0x01010101u, acc);
                v[k] = acc;
            }
            if constexpr (OB == 2) {
#pragma unroll
                for (int i = 0; i < 4; ++i) o[i] = v[2 * i] | v[2 * i + 1] << 16;
            } else {
#pragma unroll
                for (int i = 0; i < 4; ++i) o[i] = v[4 * i] | v[4 * i + 1] << 8 | v[4 * i + 2] << 16 | v[4 * i + 3] << 24;
            }
        }
        *reinterpret_cast<uint4 *>(orow + (head + q * NO) * OB) = make_uint4(o[0], o[1], o[2], o[3]);
    }
    if (blockIdx.x % nchunk == 0 && threadIdx.x < 64) {  // the row's edges, one output per step
        const int64_t body_end = head + npiece * NO;
        for (int64_t k = threadIdx.x; k < head + (p.nout - body_end); k += 64) {
            const int64_t t = k < head ? k : body_end + (k - head);
            uint32_t sum = 0u;
            for (int i = 0; i < F; ++i) {
                const int64_t e = t * F + i;
                if (MODE == DD_U4) {
                    const uint32_t b = row[e >> 1];
                    sum += (e & 1) ? b >> 4 : b & 15u;
                } else {
                    sum += row[e];
                }
            }
            if (OB == 2)
                reinterpret_cast<uint16_t *>(orow)[t] = static_cast<uint16_t>(sum);
            else
                orow[t] = static_cast<uint8_t>(sum);
        }
    }
}

// float32: a thread makes four consecutive outputs from 4*F consecutive inputs, all loads first,
// each output summed in ascending i; VEC = widest vector (floats) the row alignment allows.
template <int F, int VEC>
__global__ void __launch_bounds__(256) bin_time_f32_kernel(const BinParams p)
{
    const int64_t nchunk = p.row_chunks;
    const int c = static_cast<int>(blockIdx.x / nchunk);
    const int64_t o0 = (static_cast<int64_t>(blockIdx.x % nchunk) * 256 + threadIdx.x) * 4;
    if (o0 >= p.nout) return;
    const float *row = static_cast<const float *>(p.in) + static_cast<size_t>(c) * p.nsamps + o0 * F;
    float *orow = static_cast<float *>(p.out) + static_cast<size_t>(c) * p.nout + o0;
    const int nvalid = p.nout - o0 < 4 ? static_cast<int>(p.nout - o0) : 4;
    float x[4 * F];
    if (nvalid == 4) {
        if constexpr (VEC == 4) {
#pragma unroll
            for (int k = 0; k < F; ++k) {
                const float4 v = reinterpret_cast<const float4 *>(row)[k];
                x[4 * k] = v.x, x[4 * k + 1] = v.y, x[4 * k + 2] = v.z, x[4 * k + 3] = v.w;
            }
        } else if constexpr (VEC == 2) {
#pragma unroll
            for (int k = 0; k < 2 * F; ++k) {
                const float2 v = reinterpret_cast<const float2 *>(row)[k];
                x[2 * k] = v.x, x[2 * k + 1] = v.y;
            }
        } else {
#pragma unroll
            for (int k = 0; k < 4 * F; ++k) x[k] = row[k];
        }
    } else {
#pragma unroll
        for (int k = 0; k < 4 * F; ++k) x[k] = k < nvalid * F ? row[k] : 0.f;
    }
    float acc[4];
#pragma unroll
    for (int o = 0; o < 4; ++o) {
        acc[o] = 0.f;
#pragma unroll
        for (int i = 0; i < F; ++i) acc[o] += x[o * F + i];
    }
    if (nvalid == 4 && VEC == 4 && (reinterpret_cast<uintptr_t>(orow) & 15u) == 0) {
        *reinterpret_cast<float4 *>(orow) = make_float4(acc[0], acc[1], acc[2], acc[3]);
    } else if (nvalid == 4 && (reinterpret_cast<uintptr_t>(orow) & 7u) == 0) {
        reinterpret_cast<float2 *>(orow)[0] = make_float2(acc[0], acc[1]);
        reinterpret_cast<float2 *>(orow)[1] = make_float2(acc[2], acc[3]);
    } else {
        for (int o = 0; o < nvalid; ++o) orow[o] = acc[o];
    }
}

template <int MODE>
__global__ void __launch_bounds__(256) bin_time_kernel(const BinParams p)
{
    const int64_t nchunk = (p.nout - p.out_begin + 1023) / 1024;
    const int c = static_cast<int>(blockIdx.x / nchunk);
    const int64_t o0 = p.out_begin + (static_cast<int64_t>(blockIdx.x % nchunk) * blockDim.x + threadIdx.x) * 4;
    if (o0 >= p.nout) return;
    const int F = p.factor;
    const int nvalid = p.nout - o0 < 4 ? static_cast<int>(p.nout - o0) : 4;
    if (MODE == DD_F32) {
        const float *row = static_cast<const float *>(p.in) + static_cast<size_t>(c) * p.nsamps;
        float *orow = static_cast<float *>(p.out) + static_cast<size_t>(c) * p.nout;
        if (nvalid == 4 && (reinterpret_cast<uintptr_t>(row + o0 * F) & 15u) == 0 &&
            (reinterpret_cast<uintptr_t>(orow + o0) & 15u) == 0) {
            // 4*F consecutive floats as F float4 loads; output o owns floats [o*F, (o+1)*F),
            // summed in ascending order like the scalar path
            const float4 *v = reinterpret_cast<const float4 *>(row + o0 * F);
            float acc[4] = {0.f, 0.f, 0.f, 0.f};
            for (int k = 0; k < F; ++k) {
                const float4 x = v[k];
                const float e[4] = {x.x, x.y, x.z, x.w};
#pragma unroll
                for (int i = 0; i < 4; ++i) acc[(k * 4 + i) / F] += e[i];
            }
            *reinterpret_cast<float4 *>(orow + o0) = make_float4(acc[0], acc[1], acc[2], acc[3]);
            return;
        }
        for (int o = 0; o < nvalid; ++o) {
            float acc = 0.f;
            for (int i = 0; i < F; ++i) acc += row[(o0 + o) * F + i];
            orow[o0 + o] = acc;
        }
        return;
    }
    // integer inputs: bytes per input sample 1 (u8) or 1/2 (u4)
    const size_t row_bytes = MODE == DD_U4 ? static_cast<size_t>(p.nsamps / 2) : static_cast<size_t>(p.nsamps);
    const uint8_t *row = static_cast<const uint8_t *>(p.in) + static_cast<size_t>(c) * row_bytes;
    uint32_t sum[4] = {0u, 0u, 0u, 0u};
    const int64_t first = o0 * F;                       // first input sample of this thread
    const int bytes_per_out = MODE == DD_U4 ? F / 2 : F;  // >= 1 (F >= 2)
    const bool word_ok = nvalid == 4 && (reinterpret_cast<uintptr_t>(row) & 3u) == 0 &&
                         (bytes_per_out * 4) % 4 == 0 && ((MODE == DD_U4 ? first / 2 : first) & 3) == 0;
    if (word_ok) {
        const uint32_t *w = reinterpret_cast<const uint32_t *>(row + (MODE == DD_U4 ? first / 2 : first));
        // bytes_per_out * 4 bytes = bytes_per_out words in all; output o owns bytes
        // [o*bytes_per_out, (o+1)*bytes_per_out)
        for (int k = 0; k < bytes_per_out; ++k) {
            const uint32_t x = w[k];
#pragma unroll
            for (int b = 0; b < 4; ++b) {
                const uint32_t byte = (x >> (8 * b)) & 0xffu;
                const int o = (k * 4 + b) / bytes_per_out;
                sum[o] += MODE == DD_U4 ? (byte & 15u) + (byte >> 4) : byte;
            }
        }
    } else {
        for (int o = 0; o < nvalid; ++o)
            for (int i = 0; i < F; ++i) sum[o] += bin_sample<MODE>(row, first + static_cast<int64_t>(o) * F + i);
    }
    if (MODE == DD_U8) {
        uint16_t *orow = static_cast<uint16_t *>(p.out) + static_cast<size_t>(c) * p.nout;
        if (nvalid == 4 && (reinterpret_cast<uintptr_t>(orow + o0) & 7u) == 0) {
            *reinterpret_cast<uint2 *>(orow + o0) = make_uint2(sum[0] | sum[1] << 16, sum[2] | sum[3] << 16);
        } else {
            for (int o = 0; o < nvalid; ++o) orow[o0 + o] = static_cast<uint16_t>(sum[o]);
        }
    } else {
        uint8_t *orow = static_cast<uint8_t *>(p.out) + static_cast<size_t>(c) * p.nout;
        if (nvalid == 4 && (reinterpret_cast<uintptr_t>(orow + o0) & 3u) == 0) {
            *reinterpret_cast<uint32_t *>(orow + o0) = sum[0] | sum[1] << 8 | sum[2] << 16 | sum[3] << 24;
        } else {
            for (int o = 0; o < nvalid; ++o) orow[o0 + o] = static_cast<uint8_t>(sum[o]);
        }
    }
}

// ------------------------------------------------------------------ variant table
using KernelFn = void (*)(const KernelParams);
struct Variant {
    KernelShape shape;
    KernelFn fn;
};

#define DD_VARIANT(MODE, VW, RD, RJ, WD, WJ, CH, FM, NB, OW, TUNE)         \
    {                                                                      \
        {MODE, VW, RD, RJ, WD, WJ, CH, FM, NB, OW, TUNE},                  \
            dedisperse_kernel<MODE, VW, RD, RJ, WD, WJ, CH, FM, NB, OW>    \
    }

// Ordered per mode from the largest DM block to the smallest; dd_plan_create takes the
// first with TUNE == 0 whose shared-memory ring fits (smaller DM blocks = shorter staged
// windows; smaller CH = smaller stages).  The last rung of each mode (one DM trial per block)
// always fits.  TUNE == 1 entries exist only in tuning builds (build.py --tuning, -DDD_TUNING)
// and are reachable through the DD_FORCE_VARIANT environment variable of such a build.
// u8: LDS.64 superwords, 12 DM warps x 12 superwords, odd-lane adds on the fma pipe and the
// uint32 flush accumulators parked in tensor memory (FM = 4); profiles/r02_tuning.md.
const Variant kVariants[] = {
    //         mode  VW RD RJ  WD  WJ  CH FM NB OW tune
    DD_VARIANT(DD_U8, 2, 1, 12, 12, 1, 16, 4, 1, 4, 0),  // 0
    DD_VARIANT(DD_U8, 2, 1, 12, 12, 1, 8, 4, 1, 4, 0),   // 1
    DD_VARIANT(DD_U8, 2, 1, 12, 6, 2, 8, 4, 1, 4, 0),    // 2
    DD_VARIANT(DD_U8, 2, 1, 12, 3, 4, 4, 4, 1, 4, 0),    // 3
    DD_VARIANT(DD_U8, 2, 1, 6, 3, 4, 4, 4, 1, 4, 0),     // 4
    DD_VARIANT(DD_U8, 2, 1, 6, 1, 12, 4, 4, 1, 4, 0),    // 5  one DM per block: always fits
    DD_VARIANT(DD_U16, 2, 1, 8, 16, 1, 16, 0, 1, 4, 0),  // 6  LDS.64, 16 words per offset fetch
    DD_VARIANT(DD_U16, 1, 1, 8, 16, 1, 16, 0, 1, 4, 0),  // 7
    DD_VARIANT(DD_U16, 1, 1, 8, 4, 4, 16, 0, 1, 4, 0),   // 8
    DD_VARIANT(DD_U16, 1, 1, 8, 4, 4, 8, 0, 1, 4, 0),    // 9
    DD_VARIANT(DD_U16, 1, 1, 8, 1, 16, 4, 0, 1, 4, 0),   // 10 one DM per block: always fits
    DD_VARIANT(DD_F32, 1, 2, 24, 16, 1, 16, 0, 1, 2, 0), // 11 24 words per offset fetch
    DD_VARIANT(DD_F32, 1, 2, 8, 16, 1, 16, 0, 1, 2, 0),  // 12
    DD_VARIANT(DD_F32, 1, 1, 8, 16, 1, 16, 0, 1, 2, 0),  // 13
    DD_VARIANT(DD_F32, 1, 1, 8, 4, 4, 8, 0, 1, 2, 0),    // 14
    DD_VARIANT(DD_F32, 1, 1, 8, 1, 16, 4, 0, 1, 4, 0),   // 15 one DM per block: always fits
    // u4: eight 4-bit lanes per word, LDS.64 superwords of 16 samples, 11 DM warps x 8 superwords
    // (12 warps in all = 3 per scheduler: up to 168 registers, the 6 accumulator registers per word
    // need 156), odd nibbles by LOP3 + LEA.HI on the alu pipe, the whole-word add on the fma pipe
    DD_VARIANT(DD_U4, 2, 1, 8, 11, 1, 16, 4, 1, 4, 0),   // 16
    DD_VARIANT(DD_U4, 2, 1, 8, 11, 1, 8, 4, 1, 4, 0),    // 17
    DD_VARIANT(DD_U4, 2, 1, 8, 5, 2, 8, 4, 1, 4, 0),     // 18
    DD_VARIANT(DD_U4, 2, 1, 8, 3, 3, 4, 4, 1, 4, 0),     // 19
    DD_VARIANT(DD_U4, 2, 1, 4, 3, 3, 4, 4, 1, 4, 0),     // 20
    DD_VARIANT(DD_U4, 2, 1, 4, 1, 11, 4, 4, 1, 4, 0),    // 21 one DM per block: always fits
#ifdef DD_TUNING
    DD_VARIANT(DD_U4, 2, 1, 8, 12, 1, 16, 4, 1, 4, 1),   // 22 12 DM warps (128 registers: spills)
    DD_VARIANT(DD_U4, 2, 1, 8, 12, 1, 16, 2, 1, 4, 1),   // 23 SHF + LOP3, both adds on fma
    DD_VARIANT(DD_U4, 2, 1, 6, 12, 1, 16, 4, 1, 4, 1),   // 24 12 DM warps x 6 superwords
    DD_VARIANT(DD_U4, 4, 1, 4, 12, 1, 16, 4, 1, 4, 1),   // 25 LDS.128 x 4
    DD_VARIANT(DD_U4, 2, 1, 8, 12, 1, 16, 0, 1, 4, 1),   // 26 compiler's choice of shift-and-add
    DD_VARIANT(DD_U4, 2, 1, 8, 12, 1, 16, 3, 1, 4, 1),   // 27 IMAD.WIDE 64-bit whole-word sum
    DD_VARIANT(DD_U4, 2, 1, 8, 12, 1, 16, 1, 1, 4, 1),   // 28 W as IADD3
    DD_VARIANT(DD_U4, 2, 1, 9, 11, 1, 16, 4, 1, 4, 1),   // 29 11 DM warps x 9 superwords
    DD_VARIANT(DD_U8, 2, 1, 6, 12, 1, 32, 2, 1, 4, 1),   // r01b shape: accumulators in registers
    DD_VARIANT(DD_U8, 1, 1, 8, 16, 1, 16, 0, 1, 4, 1),   // r01 first shape
    DD_VARIANT(DD_U8, 2, 1, 6, 12, 1, 32, 1, 1, 4, 1),   // W on fma instead of O
    DD_VARIANT(DD_U8, 2, 1, 6, 12, 1, 32, 0, 1, 4, 1),   // all adds on alu
    DD_VARIANT(DD_U16, 1, 2, 8, 16, 1, 16, 0, 1, 4, 1),  // r01b shape: 2 DMs x 8 words
    DD_VARIANT(DD_F32, 1, 2, 8, 16, 1, 16, 0, 1, 4, 1),  // 32-bit offsets
    DD_VARIANT(DD_U8, 2, 1, 14, 12, 1, 16, 4, 1, 4, 1),  // 36 12 DM warps x 14 superwords
    DD_VARIANT(DD_U8, 2, 1, 16, 11, 1, 16, 4, 1, 4, 1),  // 37 11 DM warps x 16 superwords
    DD_VARIANT(DD_U8, 2, 1, 14, 11, 1, 16, 4, 1, 4, 1),  // 38 11 DM warps x 14 superwords
#endif
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

template <int VW>
static void launch_interleave_vw(int mode, const InterleaveParams &p, unsigned grid, cudaStream_t st)
{
    if (mode == DD_U4)
        interleave_u4_kernel<VW><<<grid, 256, 0, st>>>(p);
    else if (mode == DD_U8)
        interleave_kernel<DD_U8, VW><<<grid, 256, 0, st>>>(p);
    else if (mode == DD_U16)
        interleave_kernel<DD_U16, VW><<<grid, 256, 0, st>>>(p);
    else
        interleave_kernel<DD_F32, VW><<<grid, 256, 0, st>>>(p);
}

template <int MODE>
static void launch_bin_fast(const BinParams &p, unsigned grid, cudaStream_t st)
{
    switch (p.factor) {
    case 2: bin_time_fast_kernel<MODE, 2><<<grid, 256, 0, st>>>(p); break;
    case 4: bin_time_fast_kernel<MODE, 4><<<grid, 256, 0, st>>>(p); break;
    case 8: bin_time_fast_kernel<MODE, 8><<<grid, 256, 0, st>>>(p); break;
    default: bin_time_fast_kernel<MODE, 16><<<grid, 256, 0, st>>>(p); break;
    }
}

template <int MODE>
static void launch_bin_rows(const BinParams &p, unsigned grid, cudaStream_t st)
{
    switch (p.factor) {
    case 2: bin_time_rows_kernel<MODE, 2><<<grid, 256, 0, st>>>(p); break;
    case 4: bin_time_rows_kernel<MODE, 4><<<grid, 256, 0, st>>>(p); break;
    case 8: bin_time_rows_kernel<MODE, 8><<<grid, 256, 0, st>>>(p); break;
    default: bin_time_rows_kernel<MODE, 16><<<grid, 256, 0, st>>>(p); break;
    }
}

template <int VEC>
static void launch_bin_f32(const BinParams &p, unsigned grid, cudaStream_t st)
{
    switch (p.factor) {
    case 2: bin_time_f32_kernel<2, VEC><<<grid, 256, 0, st>>>(p); break;
    case 4: bin_time_f32_kernel<4, VEC><<<grid, 256, 0, st>>>(p); break;
    case 8: bin_time_f32_kernel<8, VEC><<<grid, 256, 0, st>>>(p); break;
    default: bin_time_f32_kernel<16, VEC><<<grid, 256, 0, st>>>(p); break;
    }
}

int launch_bin_time(int mode, const BinParams &p_in, void *stream)
{
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    BinParams p = p_in;
    p.out_begin = 0;
    p.row_chunks = 1;
    const uintptr_t ain = reinterpret_cast<uintptr_t>(p.in), aout = reinterpret_cast<uintptr_t>(p.out);
    if (mode == DD_F32) {
        if ((ain & 3u) == 0 && (aout & 3u) == 0) {
            // widest loads every row start allows: the thread's inputs start at multiples of 4*F floats
            const int vec = (ain & 15u) == 0 && p.nsamps % 4 == 0 ? 4 : ((ain & 7u) == 0 && p.nsamps % 2 == 0 ? 2 : 1);
            p.row_chunks = (p.nout + 1023) / 1024;
            const unsigned grid = static_cast<unsigned>(p.row_chunks * p.nchans);
            if (vec == 4)
                launch_bin_f32<4>(p, grid, st);
            else if (vec == 2)
                launch_bin_f32<2>(p, grid, st);
            else
                launch_bin_f32<1>(p, grid, st);
            return static_cast<int>(cudaGetLastError());
        }
    } else {
        // whole 16-byte pieces through the fast kernel when every row (input and output) is
        // suitably aligned; the generic kernel finishes the row tails (or does everything)
        const int NS = mode == DD_U4 ? 32 : 16, OB = mode == DD_U4 ? 1 : 2;
        const int NO = NS / p.factor;
        const size_t row_bytes = mode == DD_U4 ? static_cast<size_t>(p.nsamps / 2) : static_cast<size_t>(p.nsamps);
        const int ost = NO * OB;  // bytes per vector store
        const bool aligned = (ain & 15u) == 0 && row_bytes % 16 == 0 && (aout % ost) == 0 &&
                             (static_cast<size_t>(p.nout) * OB) % ost == 0;
        const int64_t npiece = p.nout / NO;
        if (aligned && npiece > 0) {
            const unsigned grid = static_cast<unsigned>((npiece + 1023) / 1024 * p.nchans);
            if (mode == DD_U8)
                launch_bin_fast<DD_U8>(p, grid, st);
            else
                launch_bin_fast<DD_U4>(p, grid, st);
            p.out_begin = npiece * NO;
        } else if ((ain & 3u) == 0 && (aout % OB) == 0 && p.nout >= 64) {
            // rows of any length: aligned output pieces from funnel-shifted input words
            const int64_t maxpiece = p.nout / (16 / OB) + 1;
            p.row_chunks = (maxpiece + 511) / 512;
            const unsigned grid = static_cast<unsigned>(p.row_chunks * p.nchans);
            if (mode == DD_U8)
                launch_bin_rows<DD_U8>(p, grid, st);
            else
                launch_bin_rows<DD_U4>(p, grid, st);
            return static_cast<int>(cudaGetLastError());
        }
    }
    if (p.out_begin < p.nout) {
        const unsigned grid = static_cast<unsigned>((p.nout - p.out_begin + 1023) / 1024 * p.nchans);
        if (mode == DD_U8)
            bin_time_kernel<DD_U8><<<grid, 256, 0, st>>>(p);
        else if (mode == DD_U4)
            bin_time_kernel<DD_U4><<<grid, 256, 0, st>>>(p);
        else
            bin_time_kernel<DD_F32><<<grid, 256, 0, st>>>(p);
    }
    return static_cast<int>(cudaGetLastError());
}

int launch_transpose(int mode, const TransposeParams &p, void *stream)
{
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (mode == DD_U4) {
        const dim3 g4(static_cast<unsigned>((p.nsamps / 2 + 127) / 128), static_cast<unsigned>((p.nchans + 255) / 256));
        transpose_u4_kernel<<<g4, 256, 0, st>>>(p);
        return static_cast<int>(cudaGetLastError());
    }
    const int P = mode == DD_U8 ? 4 : (mode == DD_U16 ? 2 : 1);
    const dim3 grid(static_cast<unsigned>((p.nsamps + 127) / 128),
                    static_cast<unsigned>((p.nchans + 32 * P - 1) / (32 * P)));
    if (mode == DD_U8)
        transpose_kernel<uint8_t><<<grid, 256, 0, st>>>(p);
    else if (mode == DD_U16)
        transpose_kernel<uint16_t><<<grid, 256, 0, st>>>(p);
    else
        transpose_kernel<uint32_t><<<grid, 256, 0, st>>>(p);
    return static_cast<int>(cudaGetLastError());
}

template <typename T>
static void launch_interleave_tm_t(int VW, const InterleaveParams &p, unsigned grid, cudaStream_t st)
{
    if (VW == 1)
        interleave_tm_kernel<T, 1><<<grid, 256, 0, st>>>(p);
    else if (VW == 2)
        interleave_tm_kernel<T, 2><<<grid, 256, 0, st>>>(p);
    else
        interleave_tm_kernel<T, 4><<<grid, 256, 0, st>>>(p);
}

// p.in is time-major [nsamps][in_pitch = nchans]; fills all Lw columns of all nrows rows of X
int launch_interleave_tm(int mode, int VW, const InterleaveParams &p, void *stream)
{
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (mode == DD_U4) {
        const int TJ4 = 256 / (VW * 8);
        const unsigned g4 = static_cast<unsigned>((p.Lw + TJ4 - 1) / TJ4 * ((p.nrows + 255) / 256));
        if (VW == 1)
            interleave_tm_u4_kernel<1><<<g4, 256, 0, st>>>(p);
        else if (VW == 2)
            interleave_tm_u4_kernel<2><<<g4, 256, 0, st>>>(p);
        else
            interleave_tm_u4_kernel<4><<<g4, 256, 0, st>>>(p);
        return static_cast<int>(cudaGetLastError());
    }
    const int E = mode == DD_U8 ? 1 : (mode == DD_U16 ? 2 : 4);
    const int TC = 128 / E;
    const int NL = VW * (4 / E), TJ = NL > 8 ? 16 : 32;
    const unsigned grid = static_cast<unsigned>((p.Lw + TJ - 1) / TJ * ((p.nrows + TC - 1) / TC));
    if (mode == DD_U8)
        launch_interleave_tm_t<uint8_t>(VW, p, grid, st);
    else if (mode == DD_U16)
        launch_interleave_tm_t<uint16_t>(VW, p, grid, st);
    else
        launch_interleave_tm_t<uint32_t>(VW, p, grid, st);
    return static_cast<int>(cudaGetLastError());
}

int launch_interleave(int mode, int VW, const InterleaveParams &p, void *stream)
{
    const unsigned grid = static_cast<unsigned>(static_cast<int64_t>(p.nchunk) * p.nrows);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (VW == 1)
        launch_interleave_vw<1>(mode, p, grid, st);
    else if (VW == 2)
        launch_interleave_vw<2>(mode, p, grid, st);
    else
        launch_interleave_vw<4>(mode, p, grid, st);
    return static_cast<int>(cudaGetLastError());
}

}  // namespace dd
