// dd_internal.h -- private to libdd.so.  Not part of the C ABI (that is include/dd.h) and
// shares nothing with oracle/.
#pragma once
#include <cstdint>
#include <vector>

#include "dd.h"

namespace dd {

// ---- host-side tiling of one plan --------------------------
//
// The time axis is re-indexed in "superwords" of VW 32-bit words: superword j of channel c
// carries LANES = VW * (4 | 2 | 1) samples of that channel, lane l being in[c][l*L + j]
// (word v of the superword holds lanes v*LPW .. v*LPW + LPW-1, LPW = samples per 32-bit
// word).  Every lane needs the SAME shift for a given (DM, channel), so a shifted read is a
// superword-index offset: always aligned for LDS.32/64/128, whatever the shift (DESIGN.md
// "Data layout").
struct KernelShape {
    int mode;     // DD_U8 / DD_U16 / DD_F32 / DD_U4 (eight 4-bit lanes per word)
    int VW;       // 32-bit words per superword: 1, 2, 4 (LDS.32 / LDS.64 / LDS.128)
    int RD, RJ;   // DM trials and superwords per thread
    int WD, WJ;   // consumer warps along DM and along j
    int CH;       // channels per pipeline stage (multiple of 8, <= 32)
    int FM;       // u8 / u4: which adds run as IMAD on the fma pipe (dd_kernels.cu)
    int NB;       // CTAs per SM the shared-memory ring is sized for
    int OW;       // bytes per shared-memory offset entry: 4 (byte offsets) or 2 (units of 4 bytes)
    int tune;     // 0: eligible for automatic selection; 1: DD_FORCE_VARIANT only
    int lpw() const { return mode == DD_U4 ? 8 : (mode == DD_U8 ? 4 : (mode == DD_U16 ? 2 : 1)); }
    int lanes() const { return VW * lpw(); }
    int sw_bytes() const { return VW * 4; }
    int D_DM() const { return RD * WD; }
    int D_J() const { return RJ * WJ * 32; }
    int threads() const { return (WD * WJ + 1) * 32; }  // + 1 producer warp
};

struct Tiling {
    KernelShape shape{};
    int variant = -1;          // index into the compiled kernel table
    int64_t L = 0;             // lane stride (samples), multiple of 16
    int64_t Lw = 0;            // superwords per row of the interleaved workspace X
    int nch_pad = 0;           // nchans rounded up to CH (padding rows of X stay zero)
    int ndb = 0, ntj = 0, nk = 0;  // DM blocks, j tiles, channel stages
    int panel = 1;             // DM blocks per rasterisation panel of the main kernel's grid
    int rows_bytes = 0;        // bytes of channel windows in one stage buffer (multiple of 16)
    int nstage = 0;
    int64_t smem_bytes = 0;
    int64_t stage_bytes_total = 0;  // global->shared bytes per launch (DD_INFO_STAGE_BYTES)
    // Stage k of DM block b holds the CH channels chan[k*CH .. k*CH+CH): a fixed permutation
    // that pairs short windows (high frequencies) with long ones (low frequencies) so that
    // every stage needs about the same number of bytes.
    std::vector<int32_t> chan;      // [nch_pad]            channel staged in slot k*CH + cl
    std::vector<uint8_t> ofs;       // [ndb][nk][D_DM][CH] entries of OW bytes: offset inside a stage buffer
    // [ndb][nch_pad] per slot: x = channel, y = first staged superword (16-B aligned address),
    // z = staged bytes (multiple of 16), w = byte offset of the window inside the stage buffer
    std::vector<int32_t> blk;       // 4 ints per slot
};

// Eq. 1 / Eq. 7 on the host; returns a dd_status.
int build_shift_table(int nchans, double f_high, double chan_bw, double tsamp,
                      const double *dm_list, int ndm, int32_t *table, int32_t *max_shift);

// Fill `t` for the given shape; returns false when even NSTAGE = 2 does not fit `smem_limit`.
bool build_tiling(const KernelShape &shape, int variant, const int32_t *table, int ndm,
                  int nchans, int64_t out_len, int32_t max_shift, int64_t smem_limit,
                  int num_sms, Tiling *t);

// ---- device side -------------------------------------------------------------------------
struct KernelParams {
    const uint32_t *X;
    const void *ofs;      // [ndb][nk][D_DM][CH] entries of OW bytes
    const int32_t *blk;   // 4 ints per slot (read as int4)
    void *out;
    int64_t out_len;   // valid output samples per DM row (stores are bounded by it)
    int64_t out_pitch; // elements between consecutive DM rows of `out`
    int64_t Lw;        // superwords per row of X
    int64_t L;
    int ndm, nch_pad, nk, ndb, ntj;
    int panel;         // DM blocks per rasterisation panel (1 .. ndb)
    int jt_begin;      // first j tile of this launch (the grid covers a range of tiles)
    int rows_bytes;    // channel windows of one stage; the stage's offset table follows
    int nstage;
    int stage_bytes;   // rows_bytes + D_DM*CH*OW, multiple of 16
    uint32_t one;      // 1, opaque to ptxas
};

struct InterleaveParams {
    const void *in;
    uint32_t *X;
    int64_t nsamps;    // valid samples per channel row (reads past it give 0)
    int64_t in_pitch;  // elements between consecutive channel rows of `in`
    int64_t L, Lw;
    int nchans;        // rows nchans .. nrows-1 of X are zero-filled (padding channels)
    int nrows;
    int64_t j_begin, j_end;  // superword columns [j_begin, j_end) of X to fill (multiples of 8)
    int nchunk;  // blocks per channel row: ceil((j_end - j_begin) / (SPT * 256)), a thread makes SPT = 4 (u4: 8) superwords
};

struct TransposeParams {
    const void *in;   // [nsamps][nchans]
    void *out;        // [nchans][nsamps]
    int64_t nsamps;
    int64_t nchans;
};

struct BinParams {
    const void *in;   // [nchans][nsamps]
    void *out;        // [nchans][nout], nout = nsamps / factor
    int64_t nsamps, nout;
    int64_t out_begin;  // first output column the generic kernel produces (set by launch_bin_time)
    int64_t row_chunks; // thread blocks per channel row of the row-wise kernels (set by launch_bin_time)
    int nchans, factor;
};

int num_variants();
const KernelShape &variant_shape(int v);
// cudaFuncSetAttribute(max dynamic smem) for variant v; returns cudaError_t as int.
int variant_prepare(int v, int smem_bytes);
// Launch the main kernel / the interleave pre-pass on `stream`; return cudaError_t as int.
int launch_dedisperse(int v, const KernelParams &p, int grid, int smem_bytes, void *stream);
int launch_interleave(int mode, int VW, const InterleaveParams &p, void *stream);
int launch_interleave_tm(int mode, int VW, const InterleaveParams &p, void *stream);
int launch_transpose(int mode, const TransposeParams &p, void *stream);
int launch_bin_time(int mode, const BinParams &p, void *stream);

}  // namespace dd
