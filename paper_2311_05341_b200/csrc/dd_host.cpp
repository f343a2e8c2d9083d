// dd_host.cpp -- host-only part of libdd.so: the delay table and the
// plan-time tiling metadata (a2).  No CUDA calls here; compiled with -ffp-contract=off.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <limits>

#include "dd_internal.h"

namespace dd {

namespace {
// Dispersion constant, MHz^2 s pc^-1 cm^3 (BASELINE.json north_star; reading R1).
constexpr double kDispersionConstant = 4.148808e3;

inline int64_t round_up(int64_t x, int64_t m) { return (x + m - 1) / m * m; }
}  // namespace

// Eq. 7: one coefficient per channel, scaled by each DM, divided by the
// sampling time, rounded to the nearest integer with ties to even (nearbyint under the
// default rounding mode).  Evaluated in double; the order of operations is
//   coef = C * (1/f_c^2 - 1/f_high^2);  shift = nearbyint(dm * coef / tsamp).
int build_shift_table(int nchans, double f_high, double chan_bw, double tsamp,
                      const double *dm_list, int ndm, int32_t *table, int32_t *max_shift)
{
    if (!dm_list || !table || nchans <= 0 || ndm <= 0) return DD_ERR_INVALID_ARG;
    if (!(f_high > 0.0) || !(chan_bw < 0.0) || !(tsamp > 0.0)) return DD_ERR_INVALID_ARG;
    if (!std::isfinite(f_high) || !std::isfinite(chan_bw) || !std::isfinite(tsamp))
        return DD_ERR_INVALID_ARG;
    const double f_lowest = f_high + static_cast<double>(nchans - 1) * chan_bw;
    if (!(f_lowest > 0.0)) return DD_ERR_INVALID_ARG;
    for (int d = 0; d < ndm; ++d)
        if (!std::isfinite(dm_list[d]) || dm_list[d] < 0.0) return DD_ERR_INVALID_ARG;

    std::vector<double> coef(static_cast<size_t>(nchans));
    const double inv_top = 1.0 / (f_high * f_high);
    for (int c = 0; c < nchans; ++c) {
        const double f = f_high + static_cast<double>(c) * chan_bw;
        const double inv = 1.0 / (f * f);
        coef[static_cast<size_t>(c)] = kDispersionConstant * (inv - inv_top);
    }
    int32_t biggest = 0;
    for (int d = 0; d < ndm; ++d) {
        const double dm = dm_list[d];
        int32_t *row = table + static_cast<size_t>(d) * static_cast<size_t>(nchans);
        for (int c = 0; c < nchans; ++c) {
            const double samples = dm * coef[static_cast<size_t>(c)] / tsamp;
            const double r = std::nearbyint(samples);
            if (!(r >= 0.0) || r > static_cast<double>(std::numeric_limits<int32_t>::max()))
                return DD_ERR_SHIFT_TOO_LARGE;
            const int32_t s = static_cast<int32_t>(r);
            row[c] = s;
            biggest = std::max(biggest, s);
        }
    }
    if (max_shift) *max_shift = biggest;
    return DD_OK;
}

// Plan-time tiling (the paper's T_bl / T_diff split, Eq. 6, taken from the
// exact integer table instead of two separately rounded products): per DM block and channel,
// the first staged superword (block base, aligned down to a 16-byte address for the bulk
// copy) and the staged length; per (DM, channel) the byte offset of its first superword
// inside the stage buffer.  Windows are packed back to back in a stage.
bool build_tiling(const KernelShape &shape, int variant, const int32_t *table, int ndm,
                  int nchans, int64_t out_len, int32_t max_shift, int64_t smem_limit,
                  int num_sms, Tiling *t)
{
    const int D_DM = shape.D_DM(), D_J = shape.D_J(), CH = shape.CH;
    const int S = shape.sw_bytes();  // bytes per superword
    const int A = 16 / S;            // superwords per 16 bytes (bulk-copy granule)
    t->shape = shape;
    t->variant = variant;
    t->L = round_up((out_len + shape.lanes() - 1) / shape.lanes(), 16);
    t->ntj = static_cast<int>((t->L + D_J - 1) / D_J);
    t->ndb = (ndm + D_DM - 1) / D_DM;
    t->nch_pad = static_cast<int>(round_up(nchans, CH));
    t->nk = t->nch_pad / CH;
    t->Lw = round_up(static_cast<int64_t>(t->ntj) * D_J + max_shift + 4, 8);

    // Channel permutation: slot i of the first half of each stage takes channels from the
    // top of the band (short windows), the second half mirrors them from the bottom (long
    // windows; padding channels c >= nchans count as the bottom).  Window length grows
    // almost linearly with the channel index, so every stage gets about the same bytes.
    t->chan.assign(static_cast<size_t>(t->nch_pad), 0);
    for (int k = 0; k < t->nk; ++k)
        for (int cl = 0; cl < CH; ++cl) {
            const int h = CH / 2;
            t->chan[static_cast<size_t>(k) * CH + cl] =
                cl < h ? k * h + cl : t->nch_pad - 1 - (k * h + (cl - h));
        }

    const size_t nslot = static_cast<size_t>(t->ndb) * static_cast<size_t>(t->nch_pad);
    t->blk.assign(nslot * 4, 0);
    // window sizes in int64: a coarse DM step times a long block can exceed int32, and such a
    // stage must make this rung fail (next rung: smaller DM block), never wrap around
    int64_t rows_bytes = 0;
    int64_t per_jtile_bytes = 0;
    for (int b = 0; b < t->ndb; ++b) {
        const int d0 = b * D_DM, d1 = std::min(ndm, d0 + D_DM);
        for (int k = 0; k < t->nk; ++k) {
            int64_t dst = 0;
            for (int cl = 0; cl < CH; ++cl) {
                const size_t slot = static_cast<size_t>(b) * t->nch_pad + static_cast<size_t>(k) * CH + cl;
                const int c = t->chan[static_cast<size_t>(k) * CH + cl];
                int32_t base = 0;
                int64_t sw = D_J;  // padding channel: a zero row of X, read at offset 0
                if (c < nchans) {
                    int32_t lo = std::numeric_limits<int32_t>::max(), hi = 0;
                    for (int d = d0; d < d1; ++d) {
                        const int32_t s = table[static_cast<size_t>(d) * nchans + c];
                        lo = std::min(lo, s);
                        hi = std::max(hi, s);
                    }
                    base = lo - lo % A;
                    sw = round_up(static_cast<int64_t>(D_J) + (static_cast<int64_t>(hi) - base), A);
                } else {
                    sw = round_up(D_J, A);
                }
                if (dst + sw * S > smem_limit) return false;  // this stage alone exceeds shared memory
                int32_t *q = t->blk.data() + slot * 4;
                q[0] = c;
                q[1] = base;
                q[2] = static_cast<int32_t>(sw * S);
                q[3] = static_cast<int32_t>(dst);
                dst += sw * S;
            }
            rows_bytes = std::max(rows_bytes, dst);
            per_jtile_bytes += dst;
        }
    }
    t->rows_bytes = static_cast<int>(rows_bytes);
    const int64_t ofs_stage_bytes = static_cast<int64_t>(D_DM) * CH * shape.OW;
    const int64_t stage_bytes = rows_bytes + ofs_stage_bytes;
    const int64_t barrier_bytes = 1024;  // mbarriers + slack, see dd_kernels.cu
    // NB CTAs per SM share the SM's shared memory (1 KB per CTA is reserved by the driver)
    const int64_t cta_limit = shape.NB > 1 ? (smem_limit + 1024) / shape.NB - 1024 : smem_limit;
    int nstage = static_cast<int>((cta_limit - barrier_bytes) / stage_bytes);
    nstage = std::min(nstage, std::min(8, std::max(t->nk, 2)));
    if (nstage < 2) return false;
    t->nstage = nstage;
    t->smem_bytes = barrier_bytes + nstage * stage_bytes;
    // Rasterisation panel (dd_kernels.cu): a wave of num_sms CTAs covering nb DM blocks x
    // num_sms/nb j tiles touches about nb * span + (num_sms/nb) * tile bytes of X, where tile =
    // one j tile of every channel and span = what one more DM block adds to the staged windows
    // (the shift difference across the block, summed over channels).  Minimal at
    // nb = sqrt(num_sms * tile / span) if the CTAs of a wave stay in step; they drift, and the
    // measured minimum of the DRAM traffic sits at 0.65-1.0 of that (profiles/r02_tuning.md:
    // lowfreq 8 where the model says 12, headline 15-22 for 18, c3 16 for 16), so 0.7 of it is
    // taken; panels are made equal.
    {
        // s(d,c) grows with the DM in every channel, so the rows of the largest and the smallest DM
        // bound every column; the last channel (lowest frequency, largest coefficient) tells which
        // rows those are -- dm_list need not be ascending
        int d_lo = 0, d_hi = 0;
        for (int d = 1; d < ndm; ++d) {
            const int32_t s = table[static_cast<size_t>(d) * nchans + (nchans - 1)];
            if (s < table[static_cast<size_t>(d_lo) * nchans + (nchans - 1)]) d_lo = d;
            if (s >= table[static_cast<size_t>(d_hi) * nchans + (nchans - 1)]) d_hi = d;  // ascending list: rows 0 and ndm-1
        }
        double span = 0.0;
        for (int c = 0; c < nchans; ++c)
            span += static_cast<double>(table[static_cast<size_t>(d_hi) * nchans + c] -
                                        table[static_cast<size_t>(d_lo) * nchans + c]);
        span = span * S / t->ndb;
        const double tile = static_cast<double>(t->nch_pad) * D_J * S;
        double nb = span > 0.0 ? 0.7 * std::sqrt(static_cast<double>(num_sms) * tile / span) : t->ndb;
        if (nb < 1.0) nb = 1.0;
        if (nb > t->ndb) nb = t->ndb;
        const int npanel = std::max(1, static_cast<int>(std::lround(t->ndb / nb)));
        t->panel = (t->ndb + npanel - 1) / npanel;
    }
    t->stage_bytes_total =
        (per_jtile_bytes + static_cast<int64_t>(t->ndb) * t->nk * ofs_stage_bytes) * t->ntj;

    // ofs[b][k][dl][cl] = dst(b,k,cl) + S*(s(d,c) - base(b,c)) (bytes, or /4 when OW == 2); DM rows past the end of the
    // plan repeat the block's last valid row (their results are computed and not stored).
    t->ofs.assign(static_cast<size_t>(t->ndb) * t->nk * D_DM * CH * shape.OW, 0);
    for (int b = 0; b < t->ndb; ++b)
        for (int k = 0; k < t->nk; ++k)
            for (int dl = 0; dl < D_DM; ++dl) {
                const int d = std::min(ndm - 1, b * D_DM + dl);
                uint8_t *dst = t->ofs.data() +
                               ((static_cast<size_t>(b) * t->nk + k) * D_DM + dl) * CH * shape.OW;
                for (int cl = 0; cl < CH; ++cl) {
                    const size_t slot = static_cast<size_t>(b) * t->nch_pad + static_cast<size_t>(k) * CH + cl;
                    const int32_t *q = t->blk.data() + slot * 4;
                    int32_t o = q[3];
                    if (q[0] < nchans)
                        o += S * (table[static_cast<size_t>(d) * nchans + q[0]] - q[1]);
                    if (shape.OW == 2) {  // units of 4 bytes; < 2^16 because shared memory is < 256 KB
                        const uint16_t v = static_cast<uint16_t>(o / 4);
                        std::memcpy(dst + cl * 2, &v, 2);
                    } else {
                        std::memcpy(dst + cl * 4, &o, 4);
                    }
                }
            }
    return true;
}

}  // namespace dd
