// dd_internal.h -- private to libdd.so.  Not part of the C ABI (that is include/dd.h) and
// shares nothing with oracle/.
#pragma once
#include <cstdint>
#include <vector>

#include "dd.h"

namespace dd {

// ---- host-side tiling of one plan --------------------------
//
// The time axis is re-indexed in 32-bit "words": word j of channel c carries LANES samples
// of that channel, lane k being in[c][k*L + j].  Every lane of a word needs the SAME shift
// for a given (DM, channel), so a shifted read is just a word-index offset -- no byte
// alignment problem, whatever the shift.
struct KernelShape {
    int mode;     // DD_U8 / DD_U16 / DD_F32
    int lanes;    // 4 / 2 / 1
    int RD, RW;   // DM trials and words per thread
    int WD, WJ;   // consumer warps along DM and along j
    int CH;       // channels per pipeline stage
    int D_DM() const { return RD * WD; }
    int D_J() const { return RW * WJ * 32; }
    int threads() const { return (WD * WJ + 1) * 32; }  // + 1 producer warp
};

struct Tiling {
    KernelShape shape{};
    int variant = -1;          // index into the compiled kernel table
    int64_t L = 0;             // lane stride (samples), multiple of 16
    int64_t Lw = 0;            // words per row of the interleaved workspace X
    int nch_pad = 0;           // nchans rounded up to CH (padding rows of X stay zero)
    int ndb = 0, ntj = 0, nk = 0;  // DM blocks, j tiles, channel stages
    int pitch_words = 0;       // shared-memory row pitch (words)
    int nstage = 0;
    int64_t smem_bytes = 0;
    int64_t stage_bytes_total = 0;  // global->shared bytes per launch (DD_INFO_STAGE_BYTES)
    std::vector<int32_t> ofs;       // [ndb][nk][D_DM][CH]  byte offset inside a stage buffer
    std::vector<int32_t> blk_base;  // [ndb][nch_pad]       first staged word (multiple of 4)
    std::vector<int32_t> blk_len;   // [ndb][nch_pad]       staged bytes (multiple of 16)
};

// Eq. 1 / Eq. 7 on the host; returns a dd_status.
int build_shift_table(int nchans, double f_high, double chan_bw, double tsamp,
                      const double *dm_list, int ndm, int32_t *table, int32_t *max_shift);

// Fill `t` for the given shape; returns false when even NSTAGE = 2 does not fit `smem_limit`.
bool build_tiling(const KernelShape &shape, int variant, const int32_t *table, int ndm,
                  int nchans, int64_t out_len, int32_t max_shift, int64_t smem_limit,
                  Tiling *t);

// ---- device side -------------------------------------------------------------------------
struct KernelParams {
    const uint32_t *X;
    const int32_t *ofs;
    const int32_t *blk_base;
    const int32_t *blk_len;
    void *out;
    int64_t out_len;
    int64_t Lw;
    int64_t L;
    int ndm, nch_pad, nk, ndb, ntj;
    int pitch_bytes;   // smem row pitch
    int nstage;
    int stage_bytes;   // CH*pitch_bytes + D_DM*CH*4, multiple of 16
};

struct InterleaveParams {
    const void *in;
    uint32_t *X;
    int64_t nsamps, L, Lw;
    int nchans;
    int nchunk;  // blocks per channel row: ceil(Lw / (4 * 256))
};

int num_variants();
const KernelShape &variant_shape(int v);
// cudaFuncSetAttribute(max dynamic smem) for variant v; returns cudaError_t as int.
int variant_prepare(int v, int smem_bytes);
// Launch the main kernel / the interleave pre-pass on `stream`; return cudaError_t as int.
int launch_dedisperse(int v, const KernelParams &p, int grid, int smem_bytes, void *stream);
int launch_interleave(int mode, const InterleaveParams &p, void *stream);

}  // namespace dd
