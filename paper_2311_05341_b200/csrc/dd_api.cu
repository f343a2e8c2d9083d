// dd_api.cu -- the C ABI of libdd.so (include/dd.h): plan lifetime, launches, host-buffer path.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "dd_internal.h"

struct dd_plan {
    int nchans = 0, ndm = 0, in_dtype = 0, device = -1;
    int64_t nsamps = 0, out_len = 0;
    int32_t max_shift = 0;
    double f_high = 0, chan_bw = 0, tsamp = 0;
    std::vector<double> dm_list;
    std::vector<int32_t> table;  // [ndm][nchans]
    dd::Tiling til;
    // device
    uint32_t *d_X = nullptr;
    uint8_t *d_ofs = nullptr;
    int32_t *d_blk = nullptr;
    int64_t workspace_bytes = 0;
    // dd_execute_host buffers (lazy)
    void *d_in_own = nullptr, *d_out_own = nullptr;
    static constexpr int kHostChunks = 8;
    bool host_made = false;
    int panel_override = 0;  // tuning builds: DD_PANEL
    int host_chunks = 0;  // dd_plan_set_host_chunks: 0 = default tapered schedule, n = n equal chunks
    cudaStream_t st_h2d = nullptr, st_d2h = nullptr, st_pre = nullptr, st_main2 = nullptr;
    cudaEvent_t ev_in[kHostChunks + 1] = {}, ev_done[kHostChunks + 1] = {}, ev_pre[kHostChunks + 1] = {};
    cudaEvent_t ev_out[kHostChunks + 1] = {};  // chunk g's device->host copy has finished
    int last_chunks = 0;             // chunks of the latest dd_execute_host[_tm] call
    int last_taper = 0;              // 1 if that call took the tapered schedule
    int64_t last_edge[kHostChunks + 1] = {};
    uint32_t *d_X2 = nullptr;  // second chunk workspace: chunk g+1 is interleaved while chunk g is dedispersed
    size_t x2_bytes = 0;
    // optional per-kernel timing (dd_plan_set_timing): ring of event triples
    static constexpr int kRing = 64;
    bool timing = false;
    cudaEvent_t ev[kRing][3] = {};
    bool ev_made = false;
    mutable int64_t timed_count = 0;
};

namespace {

// bytes of n consecutive samples of one channel (n even for the packed 4-bit type)
size_t sample_bytes(int dtype, int64_t n)
{
    if (dtype == DD_U4) return static_cast<size_t>(n / 2);
    return static_cast<size_t>(n) * (dtype == DD_U8 ? 1 : (dtype == DD_U16 ? 2 : 4));
}

void free_device(dd_plan *p)
{
    if (p->device >= 0) {
        int cur = -1;
        cudaGetDevice(&cur);
        if (cur != p->device) cudaSetDevice(p->device);
        cudaDeviceSynchronize();
        cudaFree(p->d_X);
        cudaFree(p->d_ofs);
        cudaFree(p->d_blk);
        cudaFree(p->d_X2);
        cudaFree(p->d_in_own);
        cudaFree(p->d_out_own);
        if (p->ev_made)
            for (auto &triple : p->ev)
                for (cudaEvent_t e : triple) cudaEventDestroy(e);
        if (p->host_made) {
            for (cudaEvent_t e : p->ev_in) cudaEventDestroy(e);
            for (cudaEvent_t e : p->ev_done) cudaEventDestroy(e);
            for (cudaEvent_t e : p->ev_pre) cudaEventDestroy(e);
            for (cudaEvent_t e : p->ev_out) cudaEventDestroy(e);
            cudaStreamDestroy(p->st_h2d);
            cudaStreamDestroy(p->st_d2h);
            cudaStreamDestroy(p->st_pre);
            cudaStreamDestroy(p->st_main2);
        }
        if (cur >= 0 && cur != p->device) cudaSetDevice(cur);
    }
}

template <typename T>
int upload(T **dst, const std::vector<T> &src)
{
    if (cudaMalloc(reinterpret_cast<void **>(dst), src.size() * sizeof(T)) != cudaSuccess) {
        cudaGetLastError();
        return DD_ERR_ALLOC;
    }
    if (cudaMemcpy(*dst, src.data(), src.size() * sizeof(T), cudaMemcpyHostToDevice) != cudaSuccess)
        return DD_ERR_CUDA;
    return DD_OK;
}

}  // namespace

extern "C" {

int dd_shift_table_build(int nchans, double f_high_MHz, double chan_bw_MHz, double tsamp_s,
                         const double *dm_list, int ndm, int32_t *table, int32_t *max_shift)
{
    return dd::build_shift_table(nchans, f_high_MHz, chan_bw_MHz, tsamp_s, dm_list, ndm, table,
                                 max_shift);
}

int dd_plan_create(dd_plan **out, int nchans, int64_t nsamps, double f_high_MHz,
                   double chan_bw_MHz, double tsamp_s, const double *dm_list, int ndm,
                   int in_dtype)
{
    if (!out) return DD_ERR_INVALID_ARG;
    *out = nullptr;
    if (!dm_list || nchans <= 0 || ndm <= 0 || nsamps <= 0) return DD_ERR_INVALID_ARG;
    if (in_dtype != DD_U8 && in_dtype != DD_U16 && in_dtype != DD_F32 && in_dtype != DD_U4)
        return DD_ERR_INVALID_ARG;
    if (in_dtype == DD_U4 && (nsamps & 1)) return DD_ERR_INVALID_ARG;  // rows are whole bytes
    // exact uint32 sums (Heimdall's overflow beyond 8192 channels)
    const uint64_t top = in_dtype == DD_U4 ? 15u : (in_dtype == DD_U8 ? 255u : 65535u);
    if (in_dtype != DD_F32 && top * static_cast<uint64_t>(nchans) >= (1ull << 32))
        return DD_ERR_OVERFLOW;

    dd_plan *p = new (std::nothrow) dd_plan;
    if (!p) return DD_ERR_ALLOC;
    int rc = DD_OK;
    try {
        p->nchans = nchans;
        p->ndm = ndm;
        p->nsamps = nsamps;
        p->in_dtype = in_dtype;
        p->f_high = f_high_MHz;
        p->chan_bw = chan_bw_MHz;
        p->tsamp = tsamp_s;
        p->dm_list.assign(dm_list, dm_list + ndm);
        p->table.resize(static_cast<size_t>(ndm) * nchans);
        rc = dd::build_shift_table(nchans, f_high_MHz, chan_bw_MHz, tsamp_s, p->dm_list.data(), ndm,
                                   p->table.data(), &p->max_shift);
        if (rc == DD_OK && p->max_shift >= nsamps) rc = DD_ERR_SHIFT_TOO_LARGE;
        if (rc != DD_OK) {
            delete p;
            return rc;
        }
        p->out_len = nsamps - p->max_shift;

        // ---- device
        int dev = -1;
        cudaDeviceProp prop;
        if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) {
            cudaGetLastError();
            delete p;
            return DD_ERR_CUDA;
        }
        if (prop.major != 10) {
            delete p;
            return DD_ERR_UNSUPPORTED_DEVICE;
        }
        p->device = dev;
        const int64_t smem_limit = static_cast<int64_t>(prop.sharedMemPerBlockOptin);

        // first compiled variant of this dtype whose shared-memory ring fits
        bool found = false;
#ifdef DD_TUNING
        const char *force = std::getenv("DD_FORCE_VARIANT");  // tuning builds only (build.py --tuning)
        const int forced = force ? std::atoi(force) : -1;
        if (const char *pe = std::getenv("DD_PANEL")) p->panel_override = std::atoi(pe);
#else
        const int forced = -1;
#endif
        for (int v = 0; v < dd::num_variants() && !found; ++v) {
            const dd::KernelShape &sh = dd::variant_shape(v);
            if (sh.mode != in_dtype) continue;
            if (forced >= 0 ? v != forced : sh.tune != 0) continue;
            found = dd::build_tiling(sh, v, p->table.data(), ndm, nchans, p->out_len, p->max_shift,
                                     smem_limit, prop.multiProcessorCount, &p->til);
        }
        if (!found) {
            p->device = -1;
            delete p;
            return DD_ERR_UNSUPPORTED_PLAN;
        }
        const dd::Tiling &t = p->til;
        // the attribute is per kernel function, not per plan: always raise it to the device limit
        // so that plans of one shape with different ring sizes can coexist
        if (dd::variant_prepare(t.variant, static_cast<int>(smem_limit)) != 0) rc = DD_ERR_CUDA;
        const size_t xbytes = static_cast<size_t>(t.nch_pad) * t.Lw * t.shape.sw_bytes();
        if (rc == DD_OK && cudaMalloc(reinterpret_cast<void **>(&p->d_X), xbytes) != cudaSuccess) {
            cudaGetLastError();
            rc = DD_ERR_ALLOC;
        }
        // padding channel rows stay zero for the life of the plan
        if (rc == DD_OK && cudaMemset(p->d_X, 0, xbytes) != cudaSuccess) rc = DD_ERR_CUDA;
        if (rc == DD_OK) rc = upload(&p->d_ofs, t.ofs);
        if (rc == DD_OK) rc = upload(&p->d_blk, t.blk);
        if (rc == DD_OK && cudaDeviceSynchronize() != cudaSuccess) rc = DD_ERR_CUDA;
        p->workspace_bytes = static_cast<int64_t>(xbytes) +
                             static_cast<int64_t>(t.ofs.size() + t.blk.size() * 4);
        // the host copies of the tiling tables are no longer needed
        std::vector<uint8_t>().swap(p->til.ofs);
        std::vector<int32_t>().swap(p->til.blk);
    } catch (const std::bad_alloc &) {
        rc = DD_ERR_ALLOC;
    }
    if (rc != DD_OK) {
        cudaGetLastError();
        free_device(p);
        delete p;
        return rc;
    }
    *out = p;
    return DD_OK;
}

int dd_plan_shift_table(const dd_plan *plan, const int32_t **table, int64_t *out_len,
                        int32_t *max_shift)
{
    if (!plan) return DD_ERR_INVALID_ARG;
    if (table) *table = plan->table.data();
    if (out_len) *out_len = plan->out_len;
    if (max_shift) *max_shift = plan->max_shift;
    return DD_OK;
}

}  // extern "C"

namespace {

// One launch pair over a block of `nsamps` input samples per channel producing `out_len`
// output samples per DM trial: the whole plan (dd_execute) or one time chunk of it
// (dd_execute_host).  The tiling tables do not depend on the block length, only L, the
// number of j tiles and the workspace row length do.
struct BlockGeom {
    int64_t nsamps, out_len;  // valid input / output samples of this block
    int64_t L, Lw;
    int ntj;
};

BlockGeom geom_for(const dd_plan *plan, int64_t out_len, int64_t nsamps)
{
    const dd::Tiling &t = plan->til;
    BlockGeom g;
    g.nsamps = nsamps;
    g.out_len = out_len;
    const int NL = t.shape.lanes();
    g.L = ((out_len + NL - 1) / NL + 15) / 16 * 16;
    g.ntj = static_cast<int>((g.L + t.shape.D_J() - 1) / t.shape.D_J());
    g.Lw = (static_cast<int64_t>(g.ntj) * t.shape.D_J() + plan->max_shift + 4 + 7) / 8 * 8;
    return g;
}

int launch_prepass(const dd_plan *plan, const BlockGeom &g, const void *d_in, int64_t in_pitch,
                   uint32_t *X, cudaStream_t st, bool time_major)
{
    const dd::Tiling &t = plan->til;
    dd::InterleaveParams ip;
    ip.in = d_in;
    ip.X = X;
    ip.nsamps = g.nsamps;
    ip.in_pitch = in_pitch;
    ip.L = g.L;
    ip.Lw = g.Lw;
    ip.nchans = plan->nchans;
    ip.nrows = t.nch_pad;
    ip.j_begin = 0;
    ip.j_end = g.Lw;
    const int spt = plan->in_dtype == DD_U4 ? 8 : 4;  // superwords per pre-pass thread
    ip.nchunk = static_cast<int>((g.Lw + spt * 256 - 1) / (spt * 256));
    return (time_major ? dd::launch_interleave_tm(plan->in_dtype, t.shape.VW, ip, st)
                       : dd::launch_interleave(plan->in_dtype, t.shape.VW, ip, st)) != 0
               ? DD_ERR_CUDA
               : DD_OK;
}

int launch_main(const dd_plan *plan, const BlockGeom &g, const uint32_t *X, void *d_out,
                int64_t out_pitch, cudaStream_t st)
{
    const dd::Tiling &t = plan->til;
    dd::KernelParams kp;
    kp.X = X;
    kp.ofs = plan->d_ofs;
    kp.blk = plan->d_blk;
    kp.out = d_out;
    kp.out_len = g.out_len;
    kp.out_pitch = out_pitch;
    kp.Lw = g.Lw;
    kp.L = g.L;
    kp.ndm = plan->ndm;
    kp.nch_pad = t.nch_pad;
    kp.nk = t.nk;
    kp.ndb = t.ndb;
    kp.panel = plan->panel_override > 0 ? (plan->panel_override < t.ndb ? plan->panel_override : t.ndb) : t.panel;
    kp.ntj = g.ntj;
    kp.jt_begin = 0;
    kp.rows_bytes = t.rows_bytes;
    kp.nstage = t.nstage;
    kp.stage_bytes = t.rows_bytes + t.shape.D_DM() * t.shape.CH * t.shape.OW;
    kp.one = 1u;
    const int grid = t.ndb * g.ntj;
    return dd::launch_dedisperse(t.variant, kp, grid, static_cast<int>(t.smem_bytes), st) != 0 ? DD_ERR_CUDA
                                                                                                : DD_OK;
}

// A plan's buffers, streams and events live on the device that was current at dd_plan_create; a launch
// from another current device would hand that device pointers it cannot use.  One process per GPU never
// gets here; an in-process multi-GPU caller must cudaSetDevice to the plan's device first.
bool on_plan_device(const dd_plan *plan)
{
    int cur = -1;
    return cudaGetDevice(&cur) == cudaSuccess && cur == plan->device;
}

// A host-buffer call of this plan (dd_execute_host*, possibly asynchronous and queued from another
// stream) owns the plan's workspaces and device buffers until its last copy back has finished:
// ev_out[last_chunks - 1] marks that moment.  Whatever uses them next waits for it first.  A no-op
// for plans that never took the host path (nothing is queued, no event exists yet).
void wait_for_pending_host_call(const dd_plan *plan, cudaStream_t st)
{
    if (plan->host_made && plan->last_chunks > 0)
        cudaStreamWaitEvent(st, plan->ev_out[plan->last_chunks - 1], 0);
}

int launch_block(const dd_plan *plan, const BlockGeom &g, const void *d_in, int64_t in_pitch,
                 void *d_out, int64_t out_pitch, cudaStream_t st, const cudaEvent_t *ev,
                 bool time_major = false)
{
    wait_for_pending_host_call(plan, st);
    if (ev) cudaEventRecord(ev[0], st);
    int rc = launch_prepass(plan, g, d_in, in_pitch, plan->d_X, st, time_major);
    if (rc != DD_OK) return rc;
    if (ev) cudaEventRecord(ev[1], st);
    rc = launch_main(plan, g, plan->d_X, d_out, out_pitch, st);
    if (rc != DD_OK) return rc;
    if (ev) cudaEventRecord(ev[2], st);
    return DD_OK;
}

}  // namespace

extern "C" {

int dd_execute(const dd_plan *plan, const void *d_in, void *d_out, void *cuda_stream)
{
    if (!plan || !d_in || !d_out) return DD_ERR_INVALID_ARG;
    if (!on_plan_device(plan)) return DD_ERR_INVALID_ARG;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const cudaEvent_t *ev = plan->timing ? plan->ev[plan->timed_count % dd_plan::kRing] : nullptr;
    const BlockGeom g = geom_for(plan, plan->out_len, plan->nsamps);
    const int rc = launch_block(plan, g, d_in, plan->nsamps, d_out, plan->out_len, st, ev);
    if (rc == DD_OK && ev) ++plan->timed_count;
    return rc;
}

int dd_execute_tm(const dd_plan *plan, const void *d_in_tm, void *d_out, void *cuda_stream)
{
    if (!plan || !d_in_tm || !d_out) return DD_ERR_INVALID_ARG;
    if (plan->in_dtype == DD_U4 && (plan->nchans & 1)) return DD_ERR_UNSUPPORTED_PLAN;  // whole bytes per time row
    if (!on_plan_device(plan)) return DD_ERR_INVALID_ARG;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const cudaEvent_t *ev = plan->timing ? plan->ev[plan->timed_count % dd_plan::kRing] : nullptr;
    const BlockGeom g = geom_for(plan, plan->out_len, plan->nsamps);
    // in_pitch = elements per TIME row of the time-major block
    const int rc = launch_block(plan, g, d_in_tm, plan->nchans, d_out, plan->out_len, st, ev, true);
    if (rc == DD_OK && ev) ++plan->timed_count;
    return rc;
}

int dd_transpose(const void *d_in_tm, void *d_out, int nchans, int64_t nsamps, int dtype,
                 void *cuda_stream)
{
    if (!d_in_tm || !d_out || nchans <= 0 || nsamps <= 0) return DD_ERR_INVALID_ARG;
    if (dtype != DD_U8 && dtype != DD_U16 && dtype != DD_F32 && dtype != DD_U4) return DD_ERR_INVALID_ARG;
    if (dtype == DD_U4 && ((nchans & 1) || (nsamps & 1))) return DD_ERR_INVALID_ARG;  // whole bytes both ways
    dd::TransposeParams tp;
    tp.in = d_in_tm;
    tp.out = d_out;
    tp.nsamps = nsamps;
    tp.nchans = nchans;
    return dd::launch_transpose(dtype, tp, cuda_stream) == 0 ? DD_OK : DD_ERR_CUDA;
}

int dd_bin_time(const void *d_in, void *d_out, int nchans, int64_t nsamps, int factor, int in_dtype,
                void *cuda_stream)
{
    if (!d_in || !d_out || nchans <= 0 || nsamps <= 0) return DD_ERR_INVALID_ARG;
    if (factor != 2 && factor != 4 && factor != 8 && factor != 16) return DD_ERR_INVALID_ARG;
    if (in_dtype == DD_U16) return DD_ERR_UNSUPPORTED_PLAN;  // no wider integer input type to bin into
    if (in_dtype != DD_U8 && in_dtype != DD_F32 && in_dtype != DD_U4) return DD_ERR_INVALID_ARG;
    if (in_dtype == DD_U4 && (nsamps & 1)) return DD_ERR_INVALID_ARG;
    if (nsamps / factor == 0) return DD_ERR_INVALID_ARG;
    dd::BinParams bp;
    bp.in = d_in;
    bp.out = d_out;
    bp.nsamps = nsamps;
    bp.nout = nsamps / factor;
    bp.nchans = nchans;
    bp.factor = factor;
    return dd::launch_bin_time(in_dtype, bp, cuda_stream) == 0 ? DD_OK : DD_ERR_CUDA;
}

int dd_plan_set_timing(dd_plan *plan, int on)
{
    if (!plan) return DD_ERR_INVALID_ARG;
    if (on && !plan->ev_made) {
        for (auto &triple : plan->ev)
            for (cudaEvent_t &e : triple)
                if (cudaEventCreate(&e) != cudaSuccess) return DD_ERR_CUDA;
        plan->ev_made = true;
    }
    plan->timing = on != 0;
    return DD_OK;
}

int dd_plan_kernel_times(dd_plan *plan, int max_n, float *interleave_ms, float *main_ms)
{
    if (!plan || max_n < 0) return DD_ERR_INVALID_ARG;
    int64_t n = plan->timed_count < dd_plan::kRing ? plan->timed_count : dd_plan::kRing;
    if (n > max_n) n = max_n;
    if (n == 0) return 0;
    const int64_t last = plan->timed_count - 1;
    if (cudaEventSynchronize(plan->ev[last % dd_plan::kRing][2]) != cudaSuccess) return DD_ERR_CUDA;
    for (int64_t i = 0; i < n; ++i) {
        const cudaEvent_t *e = plan->ev[(last - (n - 1) + i) % dd_plan::kRing];
        float a = 0.f, b = 0.f;
        if (cudaEventElapsedTime(&a, e[0], e[1]) != cudaSuccess ||
            cudaEventElapsedTime(&b, e[1], e[2]) != cudaSuccess)
            return DD_ERR_CUDA;
        if (interleave_ms) interleave_ms[i] = a;
        if (main_ms) main_ms[i] = b;
    }
    return static_cast<int>(n);
}

// Host-buffer path, pipelined over TIME CHUNKS (the time sharding of SURVEY.md 8(e) applied
// inside one GPU): chunk g produces output samples [o0, o1) of every DM trial from input
// samples [o0, o1 + max_shift) of every channel.  Its new input samples travel host->device
// on a copy stream (one strided 2-D copy: all channels x a contiguous time range) while
// chunk g-1 is interleaved and dedispersed on the caller's stream and chunk g-2's output
// columns travel device->host on a second copy stream.  PCIe is full duplex, so a step costs
// about max(H2D, kernels, D2H) plus one chunk of fill and drain instead of their sum.  The
// kernels see a chunk as a smaller block of the same plan (same shift and tiling tables).
static int execute_host_impl(dd_plan *plan, const void *h_in, void *h_out, void *cuda_stream, bool tm, bool async);

int dd_execute_host(dd_plan *plan, const void *h_in, void *h_out, void *cuda_stream)
{
    return execute_host_impl(plan, h_in, h_out, cuda_stream, false, false);
}

int dd_execute_host_tm(dd_plan *plan, const void *h_in_tm, void *h_out, void *cuda_stream)
{
    if (plan && plan->in_dtype == DD_U4 && (plan->nchans & 1)) return DD_ERR_UNSUPPORTED_PLAN;
    return execute_host_impl(plan, h_in_tm, h_out, cuda_stream, true, false);
}

int dd_execute_host_async(dd_plan *plan, const void *h_in, void *h_out, void *cuda_stream, int time_major)
{
    if (plan && time_major && plan->in_dtype == DD_U4 && (plan->nchans & 1)) return DD_ERR_UNSUPPORTED_PLAN;
    return execute_host_impl(plan, h_in, h_out, cuda_stream, time_major != 0, true);
}

// Streams and events of the host-buffer path, created on first use: all of them or none.
static int make_host_objects(dd_plan *plan)
{
    if (plan->host_made) return DD_OK;
    constexpr int NE = dd_plan::kHostChunks + 1;
    cudaStream_t s[4] = {};
    cudaEvent_t e[4 * NE] = {};
    bool ok = true;
    // (Giving the pre-pass stream the highest priority makes the pre-pass of chunk g+1 run beside
    // chunk g's main kernel instead of in its tail -- dd_plan_host_timeline shows it -- but the
    // main kernel slows down by as much: the end-to-end time did not move, so priorities are equal.)
    for (cudaStream_t &x : s) ok = ok && cudaStreamCreateWithFlags(&x, cudaStreamNonBlocking) == cudaSuccess;
    for (cudaEvent_t &x : e) ok = ok && cudaEventCreate(&x) == cudaSuccess;  // timed: dd_plan_host_timeline
    if (!ok) {
        for (cudaStream_t x : s)
            if (x) cudaStreamDestroy(x);
        for (cudaEvent_t x : e)
            if (x) cudaEventDestroy(x);
        cudaGetLastError();
        return DD_ERR_CUDA;
    }
    plan->st_h2d = s[0];
    plan->st_d2h = s[1];
    plan->st_pre = s[2];
    plan->st_main2 = s[3];
    for (int g = 0; g < NE; ++g) {
        plan->ev_in[g] = e[g];
        plan->ev_pre[g] = e[NE + g];
        plan->ev_done[g] = e[2 * NE + g];
        plan->ev_out[g] = e[3 * NE + g];
    }
    plan->host_made = true;
    return DD_OK;
}

// Chunk edges of the host-buffer path: chunk g = output samples [edge[g], edge[g+1]).  Returns
// the number of chunks (1 .. kHostChunks).  Chunk lengths are whole j tiles when the block is
// long enough, else a multiple of 16 samples per lane (keeps every chunk's rows as aligned as
// the caller's).
static int host_schedule(const dd_plan *plan, int64_t *edge, bool async, int *tapered)
{
    *tapered = 0;
    const dd::Tiling &t = plan->til;
    const int NL = t.shape.lanes();
    const int64_t tile = static_cast<int64_t>(NL) * t.shape.D_J();
    const int64_t unit = static_cast<int64_t>(NL) * 16;
    int G = 0;
    edge[0] = 0;
    // The asynchronous form is for callers that keep several blocks in flight: the neighbouring blocks
    // hide a block's first copy in and last copy out, so a few equal chunks (fewer repeated pre-pass
    // halos and partial waves) beat the taper: headline 61.4 against 62.8 ms per block, 4-bit 38.2 against
    // 40.1 (profiles/r02_tuning.md).
    // Blocks whose copies take longer than their kernels (lowfreq: 8.6 GB in for 126 ms of kernels) keep
    // the taper in both forms: there the copy engine, not the GPU, must never idle (161 against 166 ms).
    // The estimate below uses the rates measured on the B200 this library was tuned on (first-rung kernels:
    // 54 / 33 / 17 / 9 T adds/s for 4-bit / 8-bit / 16-bit / float32 input) and 50 GB/s per direction for the
    // host link (PCIe 5 x16 as measured).  It only picks between two correct schedules; on another link or
    // for a plan on a lower ladder rung dd_plan_set_host_chunks overrides it, and dd_plan_info
    // (DD_INFO_HOST_CHUNKS / DD_INFO_HOST_TAPER) reports what the latest call took.
    bool copy_bound = false;
    {
        const double adds = static_cast<double>(plan->ndm) * plan->out_len * plan->nchans;
        const double rate = plan->in_dtype == DD_U4 ? 54e12 : plan->in_dtype == DD_U8 ? 33e12 : plan->in_dtype == DD_U16 ? 17e12 : 9e12;
        const double in_b = static_cast<double>(plan->nchans) * sample_bytes(plan->in_dtype, plan->nsamps);
        const double out_b = static_cast<double>(plan->ndm) * plan->out_len * 4.0;
        copy_bound = (in_b > out_b ? in_b : out_b) / 50e9 > 0.9 * adds / rate;
    }
    if (plan->host_chunks == 0 && (!async || copy_bound) && plan->out_len >= 32 * tile) {
        // Tapered schedule: only the first chunk's host->device copy (chunk + max_shift halo) and
        // the last chunk's device->host copy are exposed, so those two chunks are small; in
        // between a chunk may grow as long as its copy hides behind the previous chunk's kernels.
        // (A finer 12-chunk geometric taper starting at one j tile measured slower -- headline
        // 70.0 ms against 68.7 ms, 4-bit 46.6 against 43.9: every extra launch pays a partial wave.)
        double frac[dd_plan::kHostChunks] = {0.04, 0.07, 0.12, 0.20, 0.25, 0.20, 0.09, 0.03};
        int nfrac = dd_plan::kHostChunks;
#ifdef DD_TUNING
        // tuning builds only: DD_HOST_TAPER="4,12,28,32,20,4" (per cent, at most kHostChunks entries)
        if (const char *e = std::getenv("DD_HOST_TAPER")) {
            int n = 0;
            double sum = 0.0, v[dd_plan::kHostChunks];
            const char *q = e;
            while (*q && n < dd_plan::kHostChunks) {
                char *end = nullptr;
                const double x = std::strtod(q, &end);
                if (end == q || !(x > 0.0) || !std::isfinite(x)) break;
                v[n++] = x;
                sum += x;
                q = *end == ',' ? end + 1 : end;
            }
            if (n > 0 && sum > 0.0) {
                for (int i = 0; i < n; ++i) frac[i] = v[i] / sum;
                nfrac = n;
            }
        }
#endif
        double cum = 0.0;
        for (int g = 0; g < nfrac; ++g) {
            cum += frac[g];
            int64_t e = g + 1 == nfrac
                            ? plan->out_len
                            : static_cast<int64_t>(cum * static_cast<double>(plan->out_len)) / tile * tile;
            if (e > plan->out_len) e = plan->out_len;
            if (e > edge[G]) edge[++G] = e;
        }
        *tapered = 1;
        return G;
    }
    int want = plan->host_chunks ? plan->host_chunks : (async ? 4 : 6);
    if (!plan->host_chunks) {  // at least 8 j tiles per chunk so that the grid still fills the GPU
        const int64_t by_tiles = plan->out_len / (8 * tile);
        if (want > by_tiles) want = static_cast<int>(by_tiles);
    }
    if (want > dd_plan::kHostChunks) want = dd_plan::kHostChunks;
    if (want < 1) want = 1;
    const int64_t q = plan->out_len >= 4 * want * tile ? tile : unit;
    const int64_t C = ((plan->out_len + want - 1) / want + q - 1) / q * q;
    while (edge[G] < plan->out_len) {
        const int64_t e = edge[G] + C < plan->out_len ? edge[G] + C : plan->out_len;
        edge[++G] = e;
    }
    return G;
}

int dd_plan_set_host_chunks(dd_plan *plan, int nchunks)
{
    if (!plan || nchunks < 0 || nchunks > dd_plan::kHostChunks) return DD_ERR_INVALID_ARG;
    plan->host_chunks = nchunks;
    return DD_OK;
}

// tm: the host block is time-major [nsamps][nchans]; a chunk's new samples are then ONE contiguous
// range of it (a plain 1-D copy) and the chunk runs through the fused time-major pre-pass.
static int execute_host_impl(dd_plan *plan, const void *h_in, void *h_out, void *cuda_stream, bool tm, bool async)
{
    if (!plan || !h_in || !h_out) return DD_ERR_INVALID_ARG;
    if (!on_plan_device(plan)) return DD_ERR_INVALID_ARG;
    const dd::Tiling &t = plan->til;
    const int dt = plan->in_dtype;
    const size_t in_bytes = static_cast<size_t>(plan->nchans) * sample_bytes(dt, plan->nsamps);
    const size_t out_bytes = static_cast<size_t>(plan->ndm) * plan->out_len * 4;
    if (!plan->d_in_own && cudaMalloc(&plan->d_in_own, in_bytes) != cudaSuccess) {
        cudaGetLastError();
        plan->d_in_own = nullptr;
        return DD_ERR_ALLOC;
    }
    if (!plan->d_out_own && cudaMalloc(&plan->d_out_own, out_bytes) != cudaSuccess) {
        cudaGetLastError();
        plan->d_out_own = nullptr;
        return DD_ERR_ALLOC;
    }
    if (const int rc = make_host_objects(plan); rc != DD_OK) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    int64_t edge[dd_plan::kHostChunks + 1];  // chunk g = output samples [edge[g], edge[g+1])
    int tapered = 0;
    const int G = host_schedule(plan, edge, async, &tapered);

    const unsigned char *hin = static_cast<const unsigned char *>(h_in);
    unsigned char *din = static_cast<unsigned char *>(plan->d_in_own);
    unsigned char *hout = static_cast<unsigned char *>(h_out);
    unsigned char *dout = static_cast<unsigned char *>(plan->d_out_own);
    const size_t in_pitch = sample_bytes(dt, plan->nsamps);
    const size_t out_pitch = static_cast<size_t>(plan->out_len) * 4;

    // second workspace, large enough for the longest chunk
    {
        size_t need_x = 0;
        for (int g = 0; g < G; ++g) {
            const BlockGeom bg = geom_for(plan, edge[g + 1] - edge[g], edge[g + 1] - edge[g] + plan->max_shift);
            const size_t b = static_cast<size_t>(t.nch_pad) * bg.Lw * t.shape.sw_bytes();
            if (b > need_x) need_x = b;
        }
        if (G > 1 && need_x > plan->x2_bytes) {
            cudaFree(plan->d_X2);
            plan->d_X2 = nullptr;
            plan->x2_bytes = 0;
            if (cudaMalloc(reinterpret_cast<void **>(&plan->d_X2), need_x) != cudaSuccess) {
                cudaGetLastError();
                return DD_ERR_ALLOC;
            }
            plan->x2_bytes = need_x;
        }
    }
    // Nothing has been queued so far.  From here on a failure must not return while copies or
    // kernels that touch the caller's buffers are still in flight: drain every stream first.
    auto fail = [&](int rc) {
        cudaStreamSynchronize(plan->st_h2d);
        cudaStreamSynchronize(plan->st_pre);
        cudaStreamSynchronize(plan->st_main2);
        cudaStreamSynchronize(st);
        cudaStreamSynchronize(plan->st_d2h);
        cudaGetLastError();
        return rc;
    };
    // An earlier host call of this plan may still be running, queued from ANOTHER stream (two
    // asynchronous calls, or a streaming caller that changed streams): it owns d_in_own, d_X / d_X2
    // and d_out_own until its last copy back.  `st` waits for that; every other stream of this call
    // starts behind ev_done[G] below, so the whole call does.
    wait_for_pending_host_call(plan, st);
    // the plan's streams start after whatever the caller has queued on `st`
    if (cudaEventRecord(plan->ev_done[G], st) != cudaSuccess) return DD_ERR_CUDA;
    cudaStreamWaitEvent(plan->st_h2d, plan->ev_done[G], 0);
    cudaStreamWaitEvent(plan->st_main2, plan->ev_done[G], 0);
    int64_t have = 0;  // input samples [0, have) of every channel are on their way to the device
    for (int g = 0; g < G; ++g) {
        const int64_t o0 = edge[g], o1 = edge[g + 1];
        const int64_t need = o1 + plan->max_shift;  // <= nsamps
        const int64_t need_c = dt == DD_U4 ? (need + 1) & ~static_cast<int64_t>(1) : need;  // whole bytes
        if (need_c > have) {
            cudaError_t ce;
            if (tm) {
                const size_t tb = sample_bytes(dt, plan->nchans);  // bytes of one time row
                ce = cudaMemcpyAsync(din + have * tb, hin + have * tb, static_cast<size_t>(need_c - have) * tb,
                                     cudaMemcpyHostToDevice, plan->st_h2d);
            } else {
                ce = cudaMemcpy2DAsync(din + sample_bytes(dt, have), in_pitch, hin + sample_bytes(dt, have),
                                       in_pitch, sample_bytes(dt, need_c - have), plan->nchans,
                                       cudaMemcpyHostToDevice, plan->st_h2d);
            }
            if (ce != cudaSuccess) return fail(DD_ERR_CUDA);
            have = need_c;
        }
        cudaEventRecord(plan->ev_in[g], plan->st_h2d);
        // pre-pass of chunk g on its own stream into workspace g & 1, as soon as its input has
        // arrived and the main kernel of chunk g-2 (the previous user of that workspace) is done:
        // it overlaps the main kernel of chunk g-1 (HBM-bound next to a shared-memory-bound kernel)
        const BlockGeom bg = geom_for(plan, o1 - o0, need - o0);
        uint32_t *Xg = (g & 1) ? plan->d_X2 : plan->d_X;
        cudaStreamWaitEvent(plan->st_pre, plan->ev_in[g], 0);
        if (g >= 2) cudaStreamWaitEvent(plan->st_pre, plan->ev_done[g - 2], 0);
        int rc = tm ? launch_prepass(plan, bg, din + o0 * sample_bytes(dt, plan->nchans), plan->nchans, Xg,
                                     plan->st_pre, true)
                    : launch_prepass(plan, bg, din + sample_bytes(dt, o0), plan->nsamps, Xg, plan->st_pre, false);
        if (rc != DD_OK) return fail(rc);
        cudaEventRecord(plan->ev_pre[g], plan->st_pre);
        // main kernels alternate between the caller's stream and a plan-owned one: chunks are
        // independent, so the last partial wave of chunk g overlaps the first wave of chunk g+1
        cudaStream_t sm = (g & 1) ? plan->st_main2 : st;
        cudaStreamWaitEvent(sm, plan->ev_pre[g], 0);
        rc = launch_main(plan, bg, Xg, dout + o0 * 4, plan->out_len, sm);
        if (rc != DD_OK) return fail(rc);
        cudaEventRecord(plan->ev_done[g], sm);
        cudaStreamWaitEvent(plan->st_d2h, plan->ev_done[g], 0);
        if (cudaMemcpy2DAsync(hout + o0 * 4, out_pitch, dout + o0 * 4, out_pitch,
                              static_cast<size_t>(o1 - o0) * 4, plan->ndm, cudaMemcpyDeviceToHost,
                              plan->st_d2h) != cudaSuccess)
            return fail(DD_ERR_CUDA);
        cudaEventRecord(plan->ev_out[g], plan->st_d2h);
    }
    plan->last_chunks = G;
    plan->last_taper = tapered;
    for (int g = 0; g <= G; ++g) plan->last_edge[g] = edge[g];
    // every main kernel precedes a copy on st_d2h; the caller's stream also waits for the odd chunks
    if (G > 1) cudaStreamWaitEvent(st, plan->ev_done[((G - 1) & 1) ? G - 1 : G - 2], 0);
    // ... and for the last copy back, so that "the caller's stream has reached this point" means
    // "h_out is complete" (what the asynchronous form promises)
    cudaStreamWaitEvent(st, plan->ev_out[G - 1], 0);
    if (async) return cudaGetLastError() == cudaSuccess ? DD_OK : fail(DD_ERR_CUDA);
    if (cudaStreamSynchronize(plan->st_d2h) != cudaSuccess) return fail(DD_ERR_CUDA);
    if (cudaStreamSynchronize(st) != cudaSuccess) return fail(DD_ERR_CUDA);
    return DD_OK;
}

int dd_plan_host_timeline(dd_plan *plan, int max_chunks, int64_t *out_begin, float *h2d_ms, float *pre_ms,
                          float *main_ms, float *d2h_ms)
{
    if (!plan || max_chunks < 0) return DD_ERR_INVALID_ARG;
    if (!plan->host_made || plan->last_chunks == 0) return 0;
    const int G = plan->last_chunks < max_chunks ? plan->last_chunks : max_chunks;
    // ev_done[last_chunks] was recorded on the caller's stream when the call started
    const cudaEvent_t t0 = plan->ev_done[plan->last_chunks];
    // (an asynchronous call may still be running: wait for its last copy back)
    if (cudaEventSynchronize(plan->ev_out[plan->last_chunks - 1]) != cudaSuccess) {
        cudaGetLastError();
        return DD_ERR_CUDA;
    }
    for (int g = 0; g < G; ++g) {
        float a = 0.f, b = 0.f, c = 0.f, d = 0.f;
        if (cudaEventElapsedTime(&a, t0, plan->ev_in[g]) != cudaSuccess ||
            cudaEventElapsedTime(&b, t0, plan->ev_pre[g]) != cudaSuccess ||
            cudaEventElapsedTime(&c, t0, plan->ev_done[g]) != cudaSuccess ||
            cudaEventElapsedTime(&d, t0, plan->ev_out[g]) != cudaSuccess) {
            cudaGetLastError();
            return DD_ERR_CUDA;
        }
        if (out_begin) out_begin[g] = plan->last_edge[g];
        if (h2d_ms) h2d_ms[g] = a;
        if (pre_ms) pre_ms[g] = b;
        if (main_ms) main_ms[g] = c;
        if (d2h_ms) d2h_ms[g] = d;
    }
    return G;
}

int64_t dd_plan_info(const dd_plan *plan, int what)
{
    if (!plan) return -1;
    const dd::Tiling &t = plan->til;
    switch (what) {
    case DD_INFO_D_DM: return t.shape.D_DM();
    case DD_INFO_D_J: return t.shape.D_J();
    case DD_INFO_LANES: return t.shape.lanes();
    case DD_INFO_L: return t.L;
    case DD_INFO_SMEM_BYTES: return t.smem_bytes;
    case DD_INFO_GRID: return static_cast<int64_t>(t.ndb) * t.ntj;
    case DD_INFO_THREADS: return t.shape.threads();
    case DD_INFO_WORKSPACE_BYTES: return plan->workspace_bytes;
    case DD_INFO_STAGE_BYTES: return t.stage_bytes_total;
    case DD_INFO_LAUNCHES: return 2;
    case DD_INFO_CH: return t.shape.CH;
    case DD_INFO_NSTAGE: return t.nstage;
    case DD_INFO_PANEL: return t.panel;
    case DD_INFO_HOST_CHUNKS: return plan->last_chunks;
    case DD_INFO_HOST_TAPER: return plan->last_taper;
    default: return -1;
    }
}

void dd_plan_destroy(dd_plan *plan)
{
    if (!plan) return;
    free_device(plan);
    delete plan;
}

const char *dd_strerror(int status)
{
    switch (status) {
    case DD_OK: return "ok";
    case DD_ERR_INVALID_ARG: return "invalid argument";
    case DD_ERR_SHIFT_TOO_LARGE: return "largest shift is not smaller than nsamps";
    case DD_ERR_OVERFLOW: return "channel sum does not fit uint32";
    case DD_ERR_ALLOC: return "allocation failed";
    case DD_ERR_CUDA: return "CUDA runtime error";
    case DD_ERR_UNSUPPORTED_DEVICE: return "current device is not sm_100";
    case DD_ERR_UNSUPPORTED_PLAN: return "staged window of one DM trial exceeds shared memory";
    case DD_ERR_STATIC_LIMIT: return "shift table larger than DD_NOALLOC_MAX_TABLE entries (dd_execute_noalloc's built-in scratch)";
    default: return "unknown status";
    }
}

const char *dd_version(void) { return "dd 0.1 sm_100a"; }

}  // extern "C"
