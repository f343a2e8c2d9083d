/*
 * dd.h -- C ABI of libdd.so: brute-force incoherent dedispersion on one B200 (sm_100a).
 *
 * What the library computes (arXiv 2311.05341; line numbers are /root/reference/PAPER.md):
 *
 *   out[d][t] = sum_{c=0}^{nchans-1} in[c][t + s(d,c)]          Eq. 3, Alg. 1 (72-76)
 *   s(d,c)    = rint( DM_d * C_DM * (1/f_c^2 - 1/f_high^2) / tsamp )   Eq. 1 (26-30), Eq. 7 (183-188)
 *   f_c       = f_high + c * chan_bw   (chan_bw < 0: channel 0 is the highest frequency)
 *   out_len   = nsamps - max_{d,c} s(d,c)   (the same for every DM trial)
 *
 * C_DM = 4148.808 MHz^2 s pc^-1 cm^3; shifts are evaluated in IEEE double, rounded
 * half-to-even.  Integer inputs (uint8, uint16) give exact uint32 sums; float32 input gives
 * float32 sums (summation order unspecified).  No division by nchans (Alg. 2's last line,
 * PAPER.md:120, is dropped).  Readings of the paper are listed in DESIGN.md.
 *
 * All functions return DD_OK (0) or a negative dd_status; none throws, none prints.
 * Pointers are HOST pointers unless the name starts with d_ (DEVICE pointer on the plan's
 * device).  The library never takes ownership of a caller's buffer.
 * There is no CPU fallback: without a CUDA device of compute capability 10.x,
 * dd_plan_create fails with DD_ERR_UNSUPPORTED_DEVICE / DD_ERR_CUDA.
 */
#ifndef DD_H_
#define DD_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dd_plan dd_plan;

/* in_dtype of dd_plan_create */
enum { DD_U8 = 0, DD_U16 = 1, DD_F32 = 2, DD_U4 = 3 };

typedef enum dd_status {
    DD_OK = 0,
    DD_ERR_INVALID_ARG = -1,        /* null pointer, non-positive size, chan_bw >= 0, bad DM ... */
    DD_ERR_SHIFT_TOO_LARGE = -2,    /* max shift >= nsamps: no output sample is complete */
    DD_ERR_OVERFLOW = -3,           /* nchans * max sample value does not fit uint32 */
    DD_ERR_ALLOC = -4,              /* host or device allocation failed */
    DD_ERR_CUDA = -5,               /* a CUDA runtime call or kernel launch failed */
    DD_ERR_UNSUPPORTED_DEVICE = -6, /* current device is not sm_100 (B200) */
    DD_ERR_UNSUPPORTED_PLAN = -7,   /* a single DM trial's staged window exceeds shared memory */
    DD_ERR_STATIC_LIMIT = -8        /* dd_execute_noalloc: ndm*nchans exceeds DD_NOALLOC_MAX_TABLE */
} dd_status;

/*
 * Host delay-table builder (Eq. 1 / Eq. 7).  Pure host code, needs
 * no GPU.  Writes table[d*nchans + c] = s(d,c) (row-major, DM major) and the largest entry
 * to *max_shift (may be NULL).
 *   nchans > 0, ndm > 0, f_high_MHz > 0, chan_bw_MHz < 0, f_high + (nchans-1)*chan_bw > 0,
 *   tsamp_s > 0, every DM finite and >= 0; otherwise DD_ERR_INVALID_ARG.
 *   A shift that does not fit int32 gives DD_ERR_SHIFT_TOO_LARGE.
 * `table` is caller-owned, ndm*nchans int32.
 */
int dd_shift_table_build(int nchans, double f_high_MHz, double chan_bw_MHz, double tsamp_s,
                         const double *dm_list, int ndm, int32_t *table, int32_t *max_shift);

/*
 * Create a plan on the CURRENT CUDA device.  Copies dm_list; builds and owns the host shift
 * table, its device-side tiling metadata and a device workspace (the lane-interleaved copy
 * of one input block).  Launches no kernel on the data path.
 *   in_dtype: DD_U8 / DD_U16 / DD_F32, or DD_U4 = packed 4-bit samples (the paper's third
 *   precision): two samples per byte, the earlier one in the low nibble,
 *   rows of nsamps/2 bytes, nsamps even; output uint32.  DD_U4 samples stay packed on chip
 *   (eight 4-bit lanes per 32-bit shared-memory word) and are summed exactly.
 * Errors (with *out = NULL): DD_ERR_INVALID_ARG (as dd_shift_table_build, plus out == NULL,
 * nsamps <= 0, unknown dtype); DD_ERR_SHIFT_TOO_LARGE (max shift >= nsamps);
 * DD_ERR_OVERFLOW (u8: 255*nchans >= 2^32; u16: 65535*nchans >= 2^32; u4: 15*nchans >= 2^32); DD_ERR_ALLOC;
 * DD_ERR_CUDA; DD_ERR_UNSUPPORTED_DEVICE; DD_ERR_UNSUPPORTED_PLAN.
 * The library reads no environment variable.  (A tuning build, `build.py --tuning`, is a separate
 * file, libdd_tuning.so: it adds the A/B kernel shapes of profiles/r02_tuning.md and honours
 * DD_FORCE_VARIANT=<n>, DD_PANEL=<n> and DD_HOST_TAPER=<per-cent list>; libdd.so never does.)
 */
int dd_plan_create(dd_plan **out, int nchans, int64_t nsamps, double f_high_MHz,
                   double chan_bw_MHz, double tsamp_s, const double *dm_list, int ndm,
                   int in_dtype);

/*
 * The plan's shift table.  *table points into plan-owned HOST memory ([ndm*nchans] int32,
 * row-major, DM major), valid until dd_plan_destroy.  Any out-pointer may be NULL.
 */
int dd_plan_shift_table(const dd_plan *plan, const int32_t **table, int64_t *out_len,
                        int32_t *max_shift);

/*
 * Run the transform (Eq. 3) once.
 *   d_in : DEVICE, dense [nchans][nsamps] of the plan's in_dtype, time contiguous
 *          (PAPER.md:114, 163-165).  Any alignment is accepted; rows that are not 4-byte
 *          aligned take a slower scalar path in the lane-interleave pre-pass.
 *   d_out: DEVICE, dense [ndm][out_len]; uint32 for DD_U8 / DD_U16, float32 for DD_F32
 *          (PAPER.md:110-115, 157).  Every element is overwritten.
 *   cuda_stream: a cudaStream_t (NULL = the legacy default stream).
 * Asynchronous on that stream: no allocation, no synchronisation, no host read of the data.
 * The plan's workspace is used by the call, so executions of ONE plan must be ordered on
 * one stream (or otherwise serialised by the caller); different plans are independent.  (One case is
 * handled for you: a dd_execute queued while a dd_execute_host_async of the same plan is pending waits
 * for that call's last copy back, whichever stream it was given.)
 * The plan belongs to the device that was current at dd_plan_create: call with that device current
 * (an in-process multi-GPU caller does cudaSetDevice first); from another device every dd_execute* and
 * dd_survey_execute* returns DD_ERR_INVALID_ARG and launches nothing.  dd_transpose, dd_bin_time and
 * dd_execute_noalloc take no plan and run on the current device.
 * Errors: DD_ERR_INVALID_ARG (null plan / pointers, wrong current device), DD_ERR_CUDA (launch failure).
 */
int dd_execute(const dd_plan *plan, const void *d_in, void *d_out, void *cuda_stream);

/*
 * The transform on TIME-MAJOR input, the order telescopes and SIGPROC filterbank files use:
 *   d_in_tm: DEVICE, dense [nsamps][nchans] of the plan's in_dtype (channel 0 = f_high).
 * The pre-pass reads the time-major block directly (a fused transpose + lane interleave: the
 * paper transposes on the GPU and counts it in its pipeline time), then the same
 * main kernel runs.  Same stream semantics, output, timing hooks and errors as dd_execute.
 * DD_U4 plans: rows of nchans/2 bytes, the EVEN channel of a byte in the low nibble; nchans must
 * be even (DD_ERR_UNSUPPORTED_PLAN otherwise).
 */
int dd_execute_tm(const dd_plan *plan, const void *d_in_tm, void *d_out, void *cuda_stream);

/*
 * Stand-alone transpose: time-major d_in_tm [nsamps][nchans] -> channel-major d_out
 * [nchans][nsamps] (the layout dd_execute, dd_execute_host and dd_bin_time take), both DEVICE,
 * dtype DD_U8 / DD_U16 / DD_F32, or DD_U4: rows of nchans/2 bytes (even channel in the low nibble) ->
 * rows of nsamps/2 bytes (earlier sample in the low nibble); nchans and nsamps even.
 * Asynchronous on the stream, no allocation.  Errors: DD_ERR_INVALID_ARG, DD_ERR_CUDA.
 */
int dd_transpose(const void *d_in_tm, void *d_out, int nchans, int64_t nsamps, int dtype,
                 void *cuda_stream);

/*
 * Time binning (downsampling), the pipeline step the paper applies per DM range before
 * dedispersion and counts in its pipeline time (Table 2's plans):
 *   out[c][t] = sum_{i < factor} in[c][factor*t + i],   t < nsamps / factor
 * (the paper gives no formula; reading R15: raw sums, a trailing partial bin is
 * dropped, integer types are widened so that the sum is exact).
 *   d_in : DEVICE, dense [nchans][nsamps] of in_dtype.
 *   d_out: DEVICE, dense [nchans][nsamps / factor]: uint16 for DD_U8, uint8 for DD_U4
 *          (unpacked: one sample per byte), float32 for DD_F32 (summed in ascending i).
 *   factor: 2, 4, 8 or 16.
 * The result is a valid input block for a plan made with tsamp*factor, nsamps/factor and the
 * output's type (DD_U16 / DD_U8 / DD_F32).  Asynchronous on the stream, no allocation.
 * Errors: DD_ERR_INVALID_ARG (nulls, sizes, factor, odd nsamps for DD_U4),
 * DD_ERR_UNSUPPORTED_PLAN (DD_U16 input: no wider integer input type), DD_ERR_CUDA.
 */
int dd_bin_time(const void *d_in, void *d_out, int nchans, int64_t nsamps, int factor, int in_dtype,
                void *cuda_stream);

/*
 * Multi-range DM survey plans: the pipeline the paper times around its dedispersion kernel --
 * optional transpose of a time-major block, time binning per DM range, dedispersion of every
 * range (Table 2, 303-309; t_c of Eq. 10 "includes the time required for
 * dedispersion, the transpose of the input data (if necessary) and downsampling", 370).
 *
 * A range is `count` DM trials dm_start + i*dm_step (one multiply, one add per trial) searched
 * on the block binned in time by bin_factor (1 = not binned; 2, 4, 8 or 16 as dd_bin_time).
 * dd_survey_create makes one dd_plan per range -- for a binned range a plan with tsamp*bin_factor,
 * nsamps/bin_factor and dd_bin_time's output type (DD_U8 -> DD_U16, DD_U4 -> DD_U8, DD_F32 ->
 * DD_F32) -- and one device buffer per distinct factor.  Errors: as dd_plan_create for any range;
 * DD_ERR_INVALID_ARG (no ranges, count <= 0, bad factor); DD_ERR_UNSUPPORTED_PLAN (a binned range
 * of DD_U16 input).  *out = NULL on error.
 *
 * dd_survey_execute: d_in DEVICE channel-major [nchans][nsamps]; d_out HOST array of nranges
 * DEVICE pointers, d_out[r] dense [count_r][out_len_r] (uint32 or float32; sizes from
 * dd_plan_shift_table(dd_survey_plan(s, r), ...)).  Bins once per distinct factor, then runs every
 * range, all asynchronously on `cuda_stream`; no allocation.
 * dd_survey_execute_tm: d_in_tm DEVICE time-major [nsamps][nchans].  Without binned ranges every
 * range reads it through the fused time-major pre-pass (dd_execute_tm); with binned ranges the
 * block is transposed once (dd_transpose, into a survey-owned buffer allocated on first use) and
 * every range reads the channel-major copy.  DD_ERR_UNSUPPORTED_PLAN for DD_U4 with an odd nchans.
 * dd_survey_plan: the plan of range r (owned by the survey; NULL if r is out of range);
 * dd_survey_range_dtype: the input type of that plan; dd_survey_num_ranges: how many.
 * dd_survey_destroy: frees everything (waits for the device); NULL is a no-op.
 */
typedef struct dd_survey dd_survey;
typedef struct dd_dm_range {
    double dm_start, dm_step;
    int32_t count;
    int32_t bin_factor;
} dd_dm_range;
int dd_survey_create(dd_survey **out, int nchans, int64_t nsamps, double f_high_MHz, double chan_bw_MHz,
                     double tsamp_s, const dd_dm_range *ranges, int nranges, int in_dtype);
int dd_survey_num_ranges(const dd_survey *survey);
const dd_plan *dd_survey_plan(const dd_survey *survey, int range);
int dd_survey_range_dtype(const dd_survey *survey, int range);
int dd_survey_execute(dd_survey *survey, const void *d_in, void *const *d_out, void *cuda_stream);
int dd_survey_execute_tm(dd_survey *survey, const void *d_in_tm, void *const *d_out, void *cuda_stream);
void dd_survey_destroy(dd_survey *survey);

/*
 * The transform (Eq. 3) without any device allocation, for small problems.
 *
 * Everything else in this header needs a plan, and dd_plan_create calls cudaMalloc.  Some callers cannot:
 * a process whose own pool already holds all of the card's memory (cudaMalloc fails there), or a real-time
 * stage that may not stall its neighbours (cudaMalloc / cudaFree synchronise the whole device).  This call
 * is for them.  It allocates nothing on the device or the host and calls no routine that does: its single
 * piece of scratch, the device copy of the shift table, is a fixed array of DD_NOALLOC_MAX_TABLE int32
 * entries (4 MiB) built into libdd.so -- every GPU that loads the library carries those 4 MiB until the
 * process exits, whether or not this call is ever made.
 *   table : HOST, int32 [ndm][nchans] row-major, every entry >= 0 -- what dd_shift_table_build writes into
 *           a buffer of the caller's; read before the call returns.
 *   d_in  : DEVICE, dense [nchans][nsamps] of in_dtype (DD_U8 / DD_U16 / DD_F32 / DD_U4, layouts as dd_execute).
 *   d_out : DEVICE, dense [ndm][out_len], out_len = nsamps - max(table); uint32, or float32 for DD_F32
 *           (channels summed in ascending order).  Every element is overwritten.
 * Runs on the CURRENT device, asynchronously on `cuda_stream`: one copy of the table into the built-in
 * array, then one kernel that reads each sample from global memory (no shared-memory tiling: expect a
 * few per cent of dd_execute's rate -- with a plan available, use the plan).
 * The first call on each device also looks up the array's device address (cudaGetSymbolAddress; nothing
 * is allocated).  Make that first call ahead of any stream capture.
 * All calls on a device share the one array, and it keeps the previous call's table: each call rewrites
 * the ndm*nchans entries it reads, so no clearing is needed, but two calls whose GPU work can overlap
 * (different streams, no ordering between them) race on it and give wrong sums.  Calls on one stream are safe.
 * Errors: DD_ERR_INVALID_ARG (nulls, sizes, dtype, a negative entry, odd nsamps for DD_U4);
 * DD_ERR_STATIC_LIMIT (ndm*nchans > DD_NOALLOC_MAX_TABLE -- nothing is launched);
 * DD_ERR_SHIFT_TOO_LARGE (max(table) >= nsamps); DD_ERR_OVERFLOW (DD_U16 with 65535*nchans >= 2^32);
 * DD_ERR_UNSUPPORTED_DEVICE (not sm_100); DD_ERR_CUDA.
 */
#define DD_NOALLOC_MAX_TABLE (1 << 20)
int dd_execute_noalloc(const int32_t *table, int ndm, int nchans, int64_t nsamps, int in_dtype,
                       const void *d_in, void *d_out, void *cuda_stream);

/*
 * The same transform with HOST buffers: h_in [nchans][nsamps], h_out [ndm][out_len].
 * Pipelined over up to 8 time chunks (the time sharding of SURVEY.md 8(e) inside one GPU): chunk g =
 * output samples [o0, o1) of every DM trial from input samples [o0, o1 + max_shift) of every
 * channel.  Default schedule: 8 tapered chunks (4, 7, 12, 20, 25, 20, 9, 3 % of the output, edges on
 * whole j tiles) when the block has at least 32 j tiles, else up to 6 equal chunks of at least 8 j
 * tiles; dd_plan_set_host_chunks overrides it.  A chunk's new input samples are copied to a
 * plan-owned device buffer on a copy stream while the previous chunk runs through the kernels
 * (pre-pass on a plan-owned stream; main kernels alternate between `cuda_stream` and a second
 * plan-owned stream so that consecutive chunks overlap at their partial last waves) and the chunk
 * before that is copied back on a second copy stream.
 * Returns after the last copy has finished.  Buffers should be page-locked for full PCIe
 * bandwidth and true overlap (pageable memory works, slower).  The device buffers, streams and
 * events are created on first use and kept until dd_plan_destroy.
 * Errors as dd_execute, plus DD_ERR_ALLOC.  On an error after work has been queued the call
 * drains every stream it used before returning, so the caller's buffers are quiescent.
 */
int dd_execute_host(dd_plan *plan, const void *h_in, void *h_out, void *cuda_stream);

/*
 * dd_execute_host for a TIME-MAJOR host block h_in_tm [nsamps][nchans] (how a telescope back
 * end or a SIGPROC file delivers it).  Same chunk pipeline; a chunk's new samples are one
 * contiguous range of the block (a plain copy instead of a strided one) and run through the
 * fused time-major pre-pass of dd_execute_tm.  Errors as dd_execute_host and dd_execute_tm.
 */
int dd_execute_host_tm(dd_plan *plan, const void *h_in_tm, void *h_out, void *cuda_stream);

/*
 * The host-buffer pipeline without the final wait: queues every copy and kernel of dd_execute_host
 * (time_major == 0) or dd_execute_host_tm (time_major != 0) and returns.  The transform is complete --
 * h_out fully written, h_in no longer read -- when `cuda_stream` reaches the point of the call (the
 * call makes that stream wait for the last copy back); both host buffers must stay valid and untouched
 * until then.  Host-buffer calls on ONE plan are serialised whatever streams they are queued from: each
 * waits for the previous one's last copy back (the plan owns one set of device buffers), and so does a
 * dd_execute / dd_execute_tm that follows a host call.  The reverse is the caller's to order: a host call
 * after a dd_execute that is still running on ANOTHER stream.  A streaming caller alternates between two plans on two streams, so that the copies of block
 * n+1 overlap the kernels of block n -- bench.py's `e2e` does exactly that.  Default schedule of this form:
 * 4 equal chunks (the neighbouring blocks hide the first copy in and the last copy out, so the taper of the
 * synchronous form is not needed) unless the block's copies take longer than its kernels (then the taper).
 * That comparison is an estimate from the rates of the machine the library was tuned on (a B200 behind a
 * 50 GB/s-per-direction host link; 54 / 33 / 17 / 9 T adds/s for 4-bit / 8-bit / 16-bit / float32 input): it
 * chooses between two correct schedules, never affects results, dd_plan_set_host_chunks overrides it and
 * dd_plan_info(DD_INFO_HOST_CHUNKS / DD_INFO_HOST_TAPER) tells which one the latest call took.
 * Errors as dd_execute_host.
 */
int dd_execute_host_async(dd_plan *plan, const void *h_in, void *h_out, void *cuda_stream, int time_major);

/*
 * Chunk count of dd_execute_host / dd_execute_host_tm for this plan: 0 = the default schedule
 * described above, 1..8 = that many equal chunks (1 = no pipelining).  DD_ERR_INVALID_ARG otherwise.
 */
int dd_plan_set_host_chunks(dd_plan *plan, int nchunks);

/*
 * Timeline of the latest dd_execute_host / dd_execute_host_tm call of this plan, for the benchmark's
 * account of the end-to-end time: for chunk g (up to max_chunks of them) the first output sample
 * out_begin[g] and the times, in milliseconds after the call started on `cuda_stream`, at which its
 * input had arrived on the device (h2d_ms), its pre-pass (pre_ms) and main kernel (main_ms) had
 * finished and its output had arrived on the host (d2h_ms); waits for that call to finish if it was an
 * asynchronous one.  Any array may be NULL.  Returns the number
 * of chunks written (0 if the plan has not run a host call), or a negative dd_status.
 */
int dd_plan_host_timeline(dd_plan *plan, int max_chunks, int64_t *out_begin, float *h2d_ms, float *pre_ms,
                          float *main_ms, float *d2h_ms);

/*
 * Facts about the plan, for tests and the benchmark.  `what` is one of DD_INFO_*; unknown
 * keys return -1.
 */
enum {
    DD_INFO_D_DM = 0,          /* DM trials per thread block */
    DD_INFO_D_J = 1,           /* superwords of the interleaved time axis per thread block */
    DD_INFO_LANES = 2,         /* samples per superword (4, 8 or 16 bytes of one channel) */
    DD_INFO_L = 3,             /* lane stride L: superword j, lane k holds in[c][k*L + j] */
    DD_INFO_SMEM_BYTES = 4,    /* dynamic shared memory per thread block */
    DD_INFO_GRID = 5,          /* thread blocks of the main kernel */
    DD_INFO_THREADS = 6,       /* threads per block of the main kernel */
    DD_INFO_WORKSPACE_BYTES = 7, /* device workspace owned by the plan */
    DD_INFO_STAGE_BYTES = 8,   /* bytes the main kernel stages global->shared per launch */
    DD_INFO_LAUNCHES = 9,      /* kernels dd_execute launches */
    DD_INFO_CH = 10,           /* channels per pipeline stage */
    DD_INFO_NSTAGE = 11,       /* pipeline stages */
    DD_INFO_PANEL = 12,        /* DM blocks per rasterisation panel of the main kernel's grid */
    DD_INFO_HOST_CHUNKS = 13,  /* time chunks of the latest dd_execute_host* call of this plan (0: none yet) */
    DD_INFO_HOST_TAPER = 14    /* 1 if that call took the tapered schedule, 0 if equal chunks */
};
int64_t dd_plan_info(const dd_plan *plan, int what);

/*
 * Per-kernel device timing for the benchmark's roofline line.  dd_plan_set_timing(plan, 1)
 * makes every later dd_execute record CUDA events around its two kernels on the launch
 * stream (a ring of the last 64 executions; a few microseconds of host time per call);
 * dd_plan_set_timing(plan, 0) stops that.  dd_plan_kernel_times waits for the most recent
 * timed execution, writes the durations (milliseconds) of up to max_n of the latest timed
 * executions, oldest first, to interleave_ms[] / main_ms[] (either may be NULL) and returns
 * how many it wrote (0 if none), or a negative dd_status.
 */
int dd_plan_set_timing(dd_plan *plan, int on);
int dd_plan_kernel_times(dd_plan *plan, int max_n, float *interleave_ms, float *main_ms);

/*
 * Measured on-chip peaks of the current device: the denominators of the benchmark's rooflines.
 * The paper derives them from data-sheet numbers (shared-memory bandwidth = 4 B x banks x clock x
 * SMs, Eq. 8; arithmetic peak, Eq. 9); this call measures them with small
 * register-only / shared-memory-only kernels, one 1024-thread CTA per SM (dd_probe.cu).
 * `what` is one of DD_PROBE_*; *value receives
 *   DD_PROBE_SM_COUNT            number of SMs
 *   DD_PROBE_SM_CLOCK_MHZ        SM clock during a probe kernel (cycle counter / CUDA-event time)
 *   DD_PROBE_LDS32/64/128        shared-memory bytes read per clock per SM with LDS.32/.64/.128
 *   DD_PROBE_IADD3 ... _SHF      lane-instructions per clock per SM of that instruction
 *                                (IADD3 = three-input integer add; VIADD16X2 = packed 2 x 16-bit add;
 *                                IMAD = 32-bit multiply-add, fma pipe; SHIFT_ADD = acc + (x >> k),
 *                                SASS LEA.HI; IMAD_HI = high half multiply-add; IDP4A = 4-way byte dot
 *                                product; LOP3, PRMT, SHF, FADD as named)
 * (A tuning build, libdd_tuning.so, compiled with -DDD_TUNING, has five more keys: the tensor-memory
 * experiments of DESIGN.md section 10, whose numbers are kept in profiles/r02_peaks.md.)
 * Blocking (synchronises the device); allocates and frees a few MB.  Errors: DD_ERR_INVALID_ARG,
 * DD_ERR_UNSUPPORTED_DEVICE, DD_ERR_ALLOC, DD_ERR_CUDA.
 */
enum {
    DD_PROBE_SM_COUNT = 0,
    DD_PROBE_SM_CLOCK_MHZ = 1,
    DD_PROBE_LDS32 = 2,
    DD_PROBE_LDS64 = 3,
    DD_PROBE_LDS128 = 4,
    DD_PROBE_IADD3 = 5,
    DD_PROBE_VIADD16X2 = 6,
    DD_PROBE_IMAD = 7,
    DD_PROBE_FADD = 8,
    DD_PROBE_LOP3 = 9,
    DD_PROBE_PRMT = 10,
    DD_PROBE_SHIFT_ADD = 11,
    DD_PROBE_IMAD_HI = 12,
    DD_PROBE_IDP4A = 13,
    DD_PROBE_SHF = 14
#ifdef DD_TUNING
    /* tensor-memory bytes per clock per SM (tcgen05.ld.32x32b.x8), alone and beside as many LDS.64 bytes;
     * float32 sample-adds per clock per SM of the accumulate loop of a "tensor memory as a second operand
     * store" kernel: operands from shared memory only, or 4 of every 8 channels through tensor-memory
     * windows (refilled / filled once) */
    ,
    DD_PROBE_TMEM_LD = 15,
    DD_PROBE_TMEM_LD_WITH_LDS = 16,
    DD_PROBE_F32_ADDS_SMEM_ONLY = 17,
    DD_PROBE_F32_ADDS_TMEM_4_OF_8 = 18,
    DD_PROBE_F32_ADDS_TMEM_4_OF_8_NO_FILL = 19
#endif
};
int dd_probe(int what, double *value);

/* Frees everything the plan owns (waits for the device first).  NULL is a no-op. */
void dd_plan_destroy(dd_plan *plan);

/* Static, never-NULL description of a dd_status value. */
const char *dd_strerror(int status);

/* Library version string, e.g. "dd 0.1 sm_100a". */
const char *dd_version(void);

#ifdef __cplusplus
}
#endif
#endif /* DD_H_ */
