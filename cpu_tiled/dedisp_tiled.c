/*
 * dedisp_tiled.c -- A STRONGER CPU BASELINE, NOT THE PRODUCT AND NOT THE ORACLE.
 *
 * The paper's CPU implementation (arXiv 2311.05341 section 3, Algorithm 2),
 * restated: loop tiling over time (D_t), DM trials (D_dm) and frequency channels (D_f),
 * OpenMP `parallel for collapse(2)` over (time tile, DM tile), the innermost D_t-long update
 * `S[:] += x[k*N_t + i + h : D_t]` vectorised by the compiler (the paper uses Cilk Plus array
 * notation with ICC; here `#pragma omp simd` with gcc).  8-bit input only,
 * as in the paper.  SURVEY.md 8(f) rank 4.
 *
 * Three deliberate differences from the printed pseudo-code:
 *   - the final `DM[...] /= channels` is dropped: raw uint32 sums (DESIGN.md
 *     reading R6), so the result can be compared bit for bit with the oracle;
 *   - h = Delta-t(j, i, k) is read from the caller's integer shift table s(d,c) instead of being
 *     evaluated in the loop (there is no t-dependence, reading R4).  The table is an input:
 *     this file contains no dispersion law;
 *   - optional (acc16 != 0, needs D_f <= 256): the channel tile's partial sum S is kept in
 *     uint16 (256 * 255 < 2^16) and widened into the uint32 plane once per (kk, j), which
 *     doubles the samples per vector add; acc16 == 0 is the printed `int S[D_t]`.
 *
 * Only tests/ (parity against oracle/) and bench.py's cpu_baseline_tiled leg may build, load
 * or call this file.  It shares no code with oracle/ or with paper_2311_05341_b200/csrc/.
 */
#include <stddef.h>
#include <stdint.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define TILED_MAX_DT 4096

/*
 * in   : [nchans][nsamps] uint8, channel-major, time contiguous
 * table: [ndm][nchans] int32 shifts, row-major
 * out  : [ndm][out_len] uint32, out_len = nsamps - max shift of the plan (reading R5)
 * D_t <= TILED_MAX_DT.  Returns 0, or -1 on a bad tile size.
 */
int tiled_dedisperse_u8(const uint8_t *in, int nchans, int64_t nsamps, const int32_t *table,
                        int ndm, int64_t out_len, uint32_t *out, int D_t, int D_dm, int D_f,
                        int acc16)
{
    if (D_t <= 0 || D_t > TILED_MAX_DT || D_dm <= 0 || D_f <= 0 || (acc16 && D_f > 256))
        return -1;
    const int64_t nti = (out_len + D_t - 1) / D_t;
    const int ndj = (ndm + D_dm - 1) / D_dm;
#pragma omp parallel for collapse(2) schedule(dynamic, 1)
    for (int64_t ti = 0; ti < nti; ti++) {          /* for i = 0 to N_t by D_t   */
        for (int tj = 0; tj < ndj; tj++) {          /* for jj = 0 to N_DM by D_dm */
            const int64_t i = ti * D_t;
            const int jj = tj * D_dm;
            const int len = (int)(out_len - i < D_t ? out_len - i : D_t);
            const int jend = jj + D_dm < ndm ? jj + D_dm : ndm;
            uint32_t S[TILED_MAX_DT];
            uint16_t S16[TILED_MAX_DT];
            for (int kk = 0; kk < nchans; kk += D_f) {   /* for kk = 0 to N_f by D_f */
                const int kend = kk + D_f < nchans ? kk + D_f : nchans;
                for (int j = jj; j < jend; j++) {
                    uint32_t *dm = out + (size_t)j * out_len + i;
                    if (acc16) {
                        for (int t = 0; t < len; t++)
                            S16[t] = 0;
                        for (int k = kk; k < kend; k++) {
                            const int32_t h = table[(size_t)j * nchans + k];
                            const uint8_t *x = in + (size_t)k * nsamps + i + h;
#pragma omp simd
                            for (int t = 0; t < len; t++)
                                S16[t] = (uint16_t)(S16[t] + x[t]);
                        }
                        if (kk == 0) {
                            for (int t = 0; t < len; t++)
                                dm[t] = S16[t];
                        } else {
                            for (int t = 0; t < len; t++)
                                dm[t] += S16[t];
                        }
                        continue;
                    }
                    if (kk == 0) {
                        for (int t = 0; t < len; t++)
                            S[t] = 0;
                    } else {
                        for (int t = 0; t < len; t++)
                            S[t] = dm[t];
                    }
                    for (int k = kk; k < kend; k++) {
                        const int32_t h = table[(size_t)j * nchans + k];
                        const uint8_t *x = in + (size_t)k * nsamps + i + h;
#pragma omp simd
                        for (int t = 0; t < len; t++)
                            S[t] += x[t];
                    }
                    for (int t = 0; t < len; t++)
                        dm[t] = S[t];
                }
            }
        }
    }
    return 0;
}

int tiled_omp_threads(void)
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
