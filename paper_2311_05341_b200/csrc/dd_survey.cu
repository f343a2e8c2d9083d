// dd_survey.cu -- multi-range DM survey plans (dd_survey_* in include/dd.h): the pipeline of the
// paper around its dedispersion kernel (Table 2, 370 Eq. 10): optional
// transpose of a time-major block, time binning per DM range, dedispersion of every range.
// Library code only drives the calls of dd_api.cu; every step runs in the kernels of
// dd_kernels.cu.
#include <cuda_runtime.h>

#include <new>
#include <vector>

#include "dd_internal.h"

struct dd_survey {
    int nchans = 0, in_dtype = 0, device = -1;
    int64_t nsamps = 0;
    std::vector<dd_plan *> plans;   // one per range
    std::vector<int> factor;        // time-binning factor of the range (1 = none)
    std::vector<int> out_dtype;     // input type of the range's plan (the binned type)
    // one binned block per distinct factor > 1, in order of first use
    std::vector<int> bin_factor;
    std::vector<void *> bin_buf;
    void *d_cm = nullptr;           // channel-major copy of a time-major block (dd_survey_execute_tm)
    size_t cm_bytes = 0;
};

namespace {

// dd_bin_time's output type (reading R15: integer sums are widened)
int binned_dtype(int in_dtype)
{
    switch (in_dtype) {
    case DD_U8: return DD_U16;
    case DD_U4: return DD_U8;
    case DD_F32: return DD_F32;
    default: return -1;  // DD_U16: no wider integer input type
    }
}

size_t block_bytes(int dtype, int nchans, int64_t nsamps)
{
    const size_t n = static_cast<size_t>(nchans) * static_cast<size_t>(nsamps);
    return dtype == DD_U4 ? n / 2 : n * (dtype == DD_U8 ? 1 : (dtype == DD_U16 ? 2 : 4));
}

// the survey's buffers and plans live on the device that was current at dd_survey_create (dd.h, dd_execute)
bool on_survey_device(const dd_survey *s)
{
    int cur = -1;
    return cudaGetDevice(&cur) == cudaSuccess && (s->device < 0 || cur == s->device);
}

void *binned_block(const dd_survey *s, int factor)
{
    for (size_t i = 0; i < s->bin_factor.size(); ++i)
        if (s->bin_factor[i] == factor) return s->bin_buf[i];
    return nullptr;
}

int run_ranges(dd_survey *s, const void *d_in_cm, const void *d_in_tm, void *const *d_out, void *stream)
{
    // time binning once per distinct factor, then every range on its block
    for (size_t i = 0; i < s->bin_factor.size(); ++i) {
        const int rc = dd_bin_time(d_in_cm, s->bin_buf[i], s->nchans, s->nsamps, s->bin_factor[i], s->in_dtype, stream);
        if (rc != DD_OK) return rc;
    }
    for (size_t r = 0; r < s->plans.size(); ++r) {
        if (!d_out[r]) return DD_ERR_INVALID_ARG;
        int rc;
        if (s->factor[r] > 1)
            rc = dd_execute(s->plans[r], binned_block(s, s->factor[r]), d_out[r], stream);
        else if (d_in_cm)
            rc = dd_execute(s->plans[r], d_in_cm, d_out[r], stream);
        else
            rc = dd_execute_tm(s->plans[r], d_in_tm, d_out[r], stream);
        if (rc != DD_OK) return rc;
    }
    return DD_OK;
}

}  // namespace

extern "C" {

int dd_survey_create(dd_survey **out, int nchans, int64_t nsamps, double f_high_MHz, double chan_bw_MHz,
                     double tsamp_s, const dd_dm_range *ranges, int nranges, int in_dtype)
{
    if (!out) return DD_ERR_INVALID_ARG;
    *out = nullptr;
    if (!ranges || nranges <= 0 || nchans <= 0 || nsamps <= 0) return DD_ERR_INVALID_ARG;
    for (int r = 0; r < nranges; ++r) {
        const int f = ranges[r].bin_factor;
        if (ranges[r].count <= 0) return DD_ERR_INVALID_ARG;
        if (f != 1 && f != 2 && f != 4 && f != 8 && f != 16) return DD_ERR_INVALID_ARG;
        if (f > 1 && binned_dtype(in_dtype) < 0) return DD_ERR_UNSUPPORTED_PLAN;
    }
    dd_survey *s = new (std::nothrow) dd_survey;
    if (!s) return DD_ERR_ALLOC;
    int rc = DD_OK;
    try {
        s->nchans = nchans;
        s->nsamps = nsamps;
        s->in_dtype = in_dtype;
        if (cudaGetDevice(&s->device) != cudaSuccess) rc = DD_ERR_CUDA;
        for (int r = 0; r < nranges && rc == DD_OK; ++r) {
            const dd_dm_range &g = ranges[r];
            std::vector<double> dms(static_cast<size_t>(g.count));
            for (int i = 0; i < g.count; ++i) dms[static_cast<size_t>(i)] = g.dm_start + static_cast<double>(i) * g.dm_step;
            const int f = g.bin_factor;
            const int dt = f == 1 ? in_dtype : binned_dtype(in_dtype);
            dd_plan *p = nullptr;
            rc = dd_plan_create(&p, nchans, nsamps / f, f_high_MHz, chan_bw_MHz, tsamp_s * static_cast<double>(f),
                                dms.data(), g.count, dt);
            if (rc != DD_OK) break;
            s->plans.push_back(p);
            s->factor.push_back(f);
            s->out_dtype.push_back(dt);
            if (f > 1 && !binned_block(s, f)) {
                void *buf = nullptr;
                if (cudaMalloc(&buf, block_bytes(dt, nchans, nsamps / f)) != cudaSuccess) {
                    cudaGetLastError();
                    rc = DD_ERR_ALLOC;
                    break;
                }
                s->bin_factor.push_back(f);
                s->bin_buf.push_back(buf);
            }
        }
    } catch (const std::bad_alloc &) {
        rc = DD_ERR_ALLOC;
    }
    if (rc != DD_OK) {
        dd_survey_destroy(s);
        return rc;
    }
    *out = s;
    return DD_OK;
}

int dd_survey_num_ranges(const dd_survey *s) { return s ? static_cast<int>(s->plans.size()) : DD_ERR_INVALID_ARG; }

const dd_plan *dd_survey_plan(const dd_survey *s, int range)
{
    if (!s || range < 0 || range >= static_cast<int>(s->plans.size())) return nullptr;
    return s->plans[static_cast<size_t>(range)];
}

int dd_survey_range_dtype(const dd_survey *s, int range)
{
    if (!s || range < 0 || range >= static_cast<int>(s->plans.size())) return DD_ERR_INVALID_ARG;
    return s->out_dtype[static_cast<size_t>(range)];
}

int dd_survey_execute(dd_survey *s, const void *d_in, void *const *d_out, void *cuda_stream)
{
    if (!s || !d_in || !d_out) return DD_ERR_INVALID_ARG;
    if (!on_survey_device(s)) return DD_ERR_INVALID_ARG;
    return run_ranges(s, d_in, nullptr, d_out, cuda_stream);
}

int dd_survey_execute_tm(dd_survey *s, const void *d_in_tm, void *const *d_out, void *cuda_stream)
{
    if (!s || !d_in_tm || !d_out) return DD_ERR_INVALID_ARG;
    if (!on_survey_device(s)) return DD_ERR_INVALID_ARG;
    if (s->bin_factor.empty())  // no binned range: every plan reads the time-major block itself
        return run_ranges(s, nullptr, d_in_tm, d_out, cuda_stream);
    // binning works on channel-major rows: transpose once (PAPER.md:370 counts it in t_c), then
    // every range -- binned or not -- reads the channel-major copy
    if (s->in_dtype == DD_U4 && (s->nchans & 1)) return DD_ERR_UNSUPPORTED_PLAN;  // whole bytes per time row
    const size_t need = block_bytes(s->in_dtype, s->nchans, s->nsamps);
    if (need > s->cm_bytes) {
        cudaFree(s->d_cm);
        s->d_cm = nullptr;
        s->cm_bytes = 0;
        if (cudaMalloc(&s->d_cm, need) != cudaSuccess) {
            cudaGetLastError();
            return DD_ERR_ALLOC;
        }
        s->cm_bytes = need;
    }
    const int rc = dd_transpose(d_in_tm, s->d_cm, s->nchans, s->nsamps, s->in_dtype, cuda_stream);
    if (rc != DD_OK) return rc;
    return run_ranges(s, s->d_cm, nullptr, d_out, cuda_stream);
}

void dd_survey_destroy(dd_survey *s)
{
    if (!s) return;
    for (dd_plan *p : s->plans) dd_plan_destroy(p);  // waits for the device
    int cur = -1;
    cudaGetDevice(&cur);
    if (s->device >= 0 && cur != s->device) cudaSetDevice(s->device);
    if (s->plans.empty()) cudaDeviceSynchronize();
    for (void *b : s->bin_buf) cudaFree(b);
    cudaFree(s->d_cm);
    if (s->device >= 0 && cur >= 0 && cur != s->device) cudaSetDevice(cur);
    delete s;
}

}  // extern "C"
