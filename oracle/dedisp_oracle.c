/*
 * dedisp_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, obviously-correct CPU statement of what the hot path of
 * arXiv 2311.05341 computes: brute-force incoherent dedispersion,
 *
 *     out[d][t] = sum_{c=0}^{nchans-1} in[c][t + s(d,c)]            (Eq. 3;
 *                                                                    PAPER.md:72-76, Alg. 1)
 *     s(d,c)    = rint( DM_d * C_DM * (1/f_c^2 - 1/f_high^2) / tsamp )  (Eq. 1;
 *                                                                    PAPER.md:183-188, Eq. 7)
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may build, load or call this file.  It shares no code, header, table or constant
 * with the CUDA library under paper_2311_05341_b200/csrc/ and neither includes the other.
 *
 * Readings of the paper adopted here (listed in DESIGN.md "Readings"):
 *   R1  C_DM = 4148.808 MHz^2 s pc^-1 cm^3 (BASELINE.json north_star; the paper prints
 *       4148.8e3 [ms], 4148.74 and 2*4148.7e3 in Eq. 1, 7, 4).
 *   R2  f_c = f_high + c*chan_bw (chan_bw < 0): channel 0 is the highest frequency and has
 *       zero delay (Eq. 7 with i = 0).
 *   R3  the real-valued delay becomes an integer sample shift by rint() under the default
 *       round-to-nearest-even mode, evaluated in double, no FMA contraction
 *       (compile with -ffp-contract=off).
 *   R4  no t-dependence in Delta-t; the sum runs over c = 0 .. nchans-1 (Eq. 3 prints N_f).
 *   R5  out_len = nsamps - max_{d,c} s(d,c), the same for every DM (Alg. 1 reads past the
 *       end of x for t near N_t; we stop where every read is in range).
 *   R6  raw sums, no division by the channel count (Alg. 2's last line is CPU-only).
 *   R7  integer inputs accumulate in uint32 (exact, order-free); float32 inputs accumulate
 *       in double, channels in ascending c, and the oracle also returns sum_c |in| for the
 *       tolerance |gpu - oracle| <= 1e-4 * sum_c |in|.
 *
 * Loop order is d, c, t with t innermost: still Alg. 1's triple loop (the three loops
 * commute for integer data; for float the c order per output is ascending either way).
 * No blocking, no fusion, no vector intrinsics.  OpenMP over d only, because this file is
 * also the timed CPU baseline.
 *
 * Pins (tests/test_oracle_pins.py, all -m "not gpu"): hand value DM=100, 1400/1500 MHz ->
 * 0.0272824109 s; printed 4-channel shift rows; half-to-even through the whole formula;
 * table invariants; closed form in[c][t] = 100c + t; DM=0 == numpy column sum; constant
 * input; single-impulse response; dispersed pulse re-aligns at its DM; literal brute force.
 * 4-bit: nibble order on a hand-written byte row; equals the u8 transform of the numpy-unpacked
 * block; literal brute force.
 */
#include <math.h>
#include <stdint.h>
#include <stddef.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_C_DM 4148.808 /* MHz^2 s pc^-1 cm^3, reading R1 */

double oracle_c_dm(void) { return ORACLE_C_DM; }

/* Eq. 1: delay in seconds between f_low and f_high (MHz) at dispersion measure dm. */
double oracle_delay_seconds(double dm, double f_low_MHz, double f_high_MHz)
{
    double k = ORACLE_C_DM * (1.0 / (f_low_MHz * f_low_MHz) - 1.0 / (f_high_MHz * f_high_MHz));
    return dm * k;
}

/* The un-rounded shift in samples, for tests that look at distance to a half-integer. */
double oracle_shift_real(double dm, double f_c_MHz, double f_high_MHz, double tsamp_s)
{
    double k = ORACLE_C_DM * (1.0 / (f_c_MHz * f_c_MHz) - 1.0 / (f_high_MHz * f_high_MHz));
    return dm * k / tsamp_s;
}

/*
 * Eq. 7 scaled by DM and divided by the sampling time, rounded (R3).
 * table is [ndm][nchans] row-major.  Returns 0, or -1 if a shift does not fit int32 / is
 * negative (chan_bw must be < 0).  *max_shift receives the largest entry.
 */
int oracle_shift_table(int nchans, double f_high_MHz, double chan_bw_MHz, double tsamp_s,
                       const double *dm_list, int ndm, int32_t *table, int32_t *max_shift)
{
    int32_t mx = 0;
    for (int d = 0; d < ndm; d++) {
        for (int c = 0; c < nchans; c++) {
            double f_c = f_high_MHz + (double)c * chan_bw_MHz; /* R2 */
            double k = ORACLE_C_DM * (1.0 / (f_c * f_c) - 1.0 / (f_high_MHz * f_high_MHz));
            double x = dm_list[d] * k / tsamp_s;
            double r = rint(x); /* R3: FE_TONEAREST, ties to even */
            if (!(r >= 0.0) || r > 2147483647.0)
                return -1;
            int32_t s = (int32_t)r;
            table[(size_t)d * nchans + c] = s;
            if (s > mx)
                mx = s;
        }
    }
    if (max_shift)
        *max_shift = mx;
    return 0;
}

/* ---- Eq. 3 / Alg. 1, integer inputs: uint32 accumulation (R7) ------------------------- */

void oracle_dedisperse_u8(const uint8_t *in, int nchans, int64_t nsamps, const int32_t *table,
                          int ndm, int64_t out_len, uint32_t *out)
{
#pragma omp parallel for schedule(dynamic, 1)
    for (int d = 0; d < ndm; d++) {
        uint32_t *o = out + (size_t)d * out_len;
        for (int64_t t = 0; t < out_len; t++)
            o[t] = 0;
        for (int c = 0; c < nchans; c++) {
            const uint8_t *x = in + (size_t)c * nsamps + table[(size_t)d * nchans + c];
            for (int64_t t = 0; t < out_len; t++)
                o[t] += x[t];
        }
    }
}

void oracle_dedisperse_u16(const uint16_t *in, int nchans, int64_t nsamps, const int32_t *table,
                           int ndm, int64_t out_len, uint32_t *out)
{
#pragma omp parallel for schedule(dynamic, 1)
    for (int d = 0; d < ndm; d++) {
        uint32_t *o = out + (size_t)d * out_len;
        for (int64_t t = 0; t < out_len; t++)
            o[t] = 0;
        for (int c = 0; c < nchans; c++) {
            const uint16_t *x = in + (size_t)c * nsamps + table[(size_t)d * nchans + c];
            for (int64_t t = 0; t < out_len; t++)
                o[t] += x[t];
        }
    }
}

/*
 * ---- packed 4-bit input (the paper's third precision) ------------
 * Reading R14: two samples per byte, the EARLIER sample in the LOW nibble
 * (sample t of a channel is nibble t & 1 of byte t >> 1 of that channel's row); rows are
 * nsamps / 2 bytes, nsamps even.  Same definition, uint32 accumulation.
 */
static uint32_t u4_sample(const uint8_t *row, int64_t t)
{
    uint8_t b = row[t >> 1];
    return (t & 1) ? (uint32_t)(b >> 4) : (uint32_t)(b & 15u);
}

void oracle_dedisperse_u4(const uint8_t *in, int nchans, int64_t nsamps, const int32_t *table,
                          int ndm, int64_t out_len, uint32_t *out)
{
#pragma omp parallel for schedule(dynamic, 1)
    for (int d = 0; d < ndm; d++) {
        uint32_t *o = out + (size_t)d * out_len;
        for (int64_t t = 0; t < out_len; t++)
            o[t] = 0;
        for (int c = 0; c < nchans; c++) {
            const uint8_t *row = in + (size_t)c * (nsamps / 2);
            int64_t s = table[(size_t)d * nchans + c];
            for (int64_t t = 0; t < out_len; t++)
                o[t] += u4_sample(row, t + s);
        }
    }
}

/*
 * ---- time binning (downsampling), a pipeline step before dedispersion --
 * Reading R15 (the paper names the step and gives no formula): out[c][t] =
 * sum_{i<factor} in[c][factor*t + i], t < nsamps / factor (a trailing partial bin is dropped),
 * raw sums like R6, the integer types widened so the sum is exact: u4 -> u8, u8 -> u16;
 * float32 stays float32 and is summed in ascending i (double here).
 * in_dtype: 0 = uint8 -> uint16 out, 2 = float32 -> double out, 3 = packed 4-bit -> uint8 out.
 */
void oracle_bin_time(const void *in, int in_dtype, int nchans, int64_t nsamps, int factor,
                     void *out)
{
    int64_t nout = nsamps / factor;
    for (int c = 0; c < nchans; c++) {
        for (int64_t t = 0; t < nout; t++) {
            if (in_dtype == 2) {
                double acc = 0.0;
                for (int i = 0; i < factor; i++)
                    acc += (double)((const float *)in)[(size_t)c * nsamps + factor * t + i];
                ((double *)out)[(size_t)c * nout + t] = acc;
            } else if (in_dtype == 0) {
                uint32_t acc = 0;
                for (int i = 0; i < factor; i++)
                    acc += ((const uint8_t *)in)[(size_t)c * nsamps + factor * t + i];
                ((uint16_t *)out)[(size_t)c * nout + t] = (uint16_t)acc;
            } else {
                uint32_t acc = 0;
                for (int i = 0; i < factor; i++)
                    acc += u4_sample((const uint8_t *)in + (size_t)c * (nsamps / 2), factor * t + i);
                ((uint8_t *)out)[(size_t)c * nout + t] = (uint8_t)acc;
            }
        }
    }
}

/* ---- float32 input: double accumulation, ascending c; also sum |in| (R7) ------------- */

void oracle_dedisperse_f32(const float *in, int nchans, int64_t nsamps, const int32_t *table,
                           int ndm, int64_t out_len, double *out, double *out_abs)
{
#pragma omp parallel for schedule(dynamic, 1)
    for (int d = 0; d < ndm; d++) {
        double *o = out + (size_t)d * out_len;
        double *a = out_abs + (size_t)d * out_len;
        for (int64_t t = 0; t < out_len; t++) {
            o[t] = 0.0;
            a[t] = 0.0;
        }
        for (int c = 0; c < nchans; c++) {
            const float *x = in + (size_t)c * nsamps + table[(size_t)d * nchans + c];
            for (int64_t t = 0; t < out_len; t++) {
                double v = (double)x[t];
                o[t] += v;
                a[t] += fabs(v);
            }
        }
    }
}

/*
 * ---- single outputs, one by one (sampled parity at full size) -------------------------
 * For point p: d = pd[p], t = pt[p]; the same definition, evaluated for that one element.
 * in_dtype: 0 = uint8, 1 = uint16, 2 = float32.  Integer results go to out_u32, float
 * results to out_f64 / out_abs (the unused ones may be NULL).
 */
void oracle_dedisperse_points(const void *in, int in_dtype, int nchans, int64_t nsamps,
                              const int32_t *table, const int32_t *pd, const int64_t *pt,
                              int64_t npoints, uint32_t *out_u32, double *out_f64, double *out_abs)
{
#pragma omp parallel for schedule(static)
    for (int64_t p = 0; p < npoints; p++) {
        const int32_t *row = table + (size_t)pd[p] * nchans;
        int64_t t = pt[p];
        if (in_dtype == 2) {
            double acc = 0.0, ab = 0.0;
            for (int c = 0; c < nchans; c++) {
                double v = (double)((const float *)in)[(size_t)c * nsamps + t + row[c]];
                acc += v;
                ab += fabs(v);
            }
            out_f64[p] = acc;
            out_abs[p] = ab;
        } else {
            uint32_t acc = 0;
            for (int c = 0; c < nchans; c++) {
                size_t i = (size_t)c * nsamps + t + row[c];
                acc += (in_dtype == 0) ? (uint32_t)((const uint8_t *)in)[i]
                                       : (uint32_t)((const uint16_t *)in)[i];
            }
            out_u32[p] = acc;
        }
    }
}

int oracle_omp_threads(void)
{
    int n = 1;
#ifdef _OPENMP
#pragma omp parallel
    {
#pragma omp master
        n = omp_get_num_threads();
    }
#endif
    return n;
}
