/*
 * ss_periodogram.h -- C ABI of the B200-native batched SuperSmoother periodogram.
 *
 * The operation is Algorithm 1 of arXiv 2111.07396 applied to every object of a
 * catalog: per (object, trial frequency) phase-fold ("t1=(tt mod p)/p"), stable sort by
 * phase, Friedman's variable-span smoother as Listing 1 states it (
 * "cross validation") or the paper's single-pass generalized-validation variant (
 * reading R12 in DESIGN.md), the chi-square statistic (reading R6) and the per-object
 * argmax.  All arithmetic is IEEE fp64 on the GPU; there is no CPU fallback.
 *
 * Frequency grid (Table 2): half-open and evenly spaced,
 *     df = (f_max - f_min) / n_freq,   f_k = f_min + k*df,   k = 0 .. n_freq-1,
 * the same grid for every object.  Ordinary (not angular) frequency in 1/[time unit].
 *
 * Catalog layout (CSR): object i owns elements [offsets[i], offsets[i+1]) of times/mags/errs, in any
 * time order.  Weights are 1/err^2.
 *
 * Periodogram value (R6):  P = (chi0 - chi2)/chi0,  chi0 = sum w (y - ybar_w)^2,
 * chi2 = sum w (y - smo)^2.  Any positive-affine variant has the same argmax.
 *
 * Degenerate cases: an object with fewer than 5 points gets a NaN row, best_freq = NaN,
 * best_index = -1.  chi0 == 0 (constant magnitudes) gives a row of zeros and best_index = 0.
 * Argmax ties resolve to the lowest index.
 *
 * Errors: every entry point returns SS_OK or an error code.  Argument errors are found before any output is
 * touched (outputs untouched); on SS_ERR_CUDA / SS_ERR_OUT_OF_MEMORY the outputs are unspecified and ss_last_error() (thread-local) describes the failure.  The library
 * never frees or retains caller memory.
 */
#ifndef SS_PERIODOGRAM_H
#define SS_PERIODOGRAM_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SS_VERSION 200 /* 0.2.0 */

typedef enum {
    SS_MODE_CROSS_VALIDATION = 0,      /* Listing 1, PAPER.md:127-297 (paper: SSO-*)            */
    SS_MODE_GENERALIZED_VALIDATION = 1 /* single-pass variant, PAPER.md:313-329 (paper: SSSP-*) */
} ss_mode_t;

typedef enum {
    SS_OK = 0,
    SS_ERR_INVALID_ARG = 1,   /* null pointer, bad sizes/grid, non-monotone offsets, non-finite data, err <= 0 */
    SS_ERR_OUT_OF_MEMORY = 2, /* workspace could not be allocated / cap too small for one tile           */
    SS_ERR_CUDA = 3,          /* a CUDA runtime call or kernel failed                                   */
    SS_ERR_UNSUPPORTED = 4    /* an object above 2^24 points, or more work items than one tile can index  */
} ss_status_t;

typedef enum { SS_PRECISION_F64 = 0, SS_PRECISION_MIXED = 1 } ss_precision_t;

/* Which kernel family serves an object (chosen by its number of points n). */
typedef enum {
    SS_PATH_AUTO = 0,
    SS_PATH_WARP = 1,  /* one warp per (object, frequency); n <= SS_WARP_MAX_N; registers + shuffles   */
    SS_PATH_BLOCK = 2, /* one CTA per (object, frequency); per-eval arrays in shared memory            */
    SS_PATH_STAGE = 3, /* one CTA per (object, frequency); per-eval arrays staged in global memory/L2  */
    SS_PATH_GROUP = 4, /* 4, 8 or 16 warps per (object, frequency); SS_WARP_MAX_N < n <= SS_GROUP_LONG_MAX_N;
                          points in registers, prefix sums in shared memory, smooths in tensor memory.
                          Beyond 2,560 points the object's y and w are read from global memory per eval    */
    SS_PATH_CLUSTER = 5 /* a thread-block cluster of 2..16 CTAs per (object, frequency); SS_GROUP_LONG_MAX_N <
                          n <= SS_CLUSTER_MAX_N; prefix sums in distributed shared memory                  */
} ss_path_t;

#define SS_WARP_MAX_N 256
#define SS_GROUP_MAX_N 2055
#define SS_GROUP_LONG_MAX_N 3584
#define SS_CLUSTER_MAX_N 40960

typedef struct {
    double alpha;           /* bass enhancement.  Default 9.0.                 */
    double span;            /* 0 = variable span (default).  In (0, 1]: Listing 1's fixed-span branch
                               (PAPER.md:202-210): one running-line smooth at this span, in both modes.
                               Served by the warp kernels for n <= SS_WARP_MAX_N, by the group kernels for
                               n <= SS_GROUP_LONG_MAX_N when span >= 0.05, by the CTA-per-eval kernels otherwise;
                               always in fp64.                                                           */
    int iper;               /* 1 = windows pinned at the ends (default, R8).  2 = periodic windows
                               (PAPER.md:199-200): the window of point j is j-ibw..j+ibw modulo n, phases
                               that wrapped count as x-1 / x+1.  Served like the fixed span (warp, group or
                               CTA-per-eval kernels by n), in fp64.                                      */
    int force_path;         /* ss_path_t; SS_PATH_AUTO = choose by n.  For tests and sweeps.            */
    void *stream;           /* cudaStream_t the work is enqueued on (NULL = legacy default stream)      */
    size_t workspace_cap;   /* bytes of device workspace the library may allocate; 0 = 75 % of free
                               device memory (the paper's beta = 0.75)                    */
    int64_t freq_tile;      /* host entry point only: force this many frequencies per output tile
                               (0 = planner decides).  For tests.                                       */
    int skip_validation;    /* 1 = trust the inputs (no device validation pass, no host sync for it)    */
    int profile;            /* 1 = bracket every eval-kernel launch with CUDA events on the stream;
                               read the sum with ss_last_kernel_ms() after the call                     */
    int64_t k_begin;        /* evaluate only the grid indices [k_begin, k_begin + k_count) of the grid that   */
    int64_t k_count;        /* (f_min, f_max, n_freq) defines: f_k keeps its bits, pgram_out then has k_count
                               columns (column 0 = index k_begin), best_index stays an index into the whole
                               grid.  k_count = 0: up to the end of the grid.  For splitting one object's
                               frequency range across GPUs.                           */
    int precision;          /* ss_precision_t.  SS_PRECISION_F64 (default): everything in fp64.  SS_PRECISION_MIXED
                               (the paper's FP32 switch): for objects of n <= SS_GROUP_LONG_MAX_N
                               points (warp and group paths, default listing options) the smoother runs in fp32 --
                               prefix arrays stored and window fits, residuals, span selection and interpolation
                               computed in float -- while the fold, the sort, the centring and the accumulation of
                               the prefix sums across threads stay in fp64 (the permutation is therefore the fp64
                               one).  Longer light curves, evals the fast path hands over (tied phases) and calls
                               with iper = 2 or a fixed span are served in fp64.  Periodogram values then agree with
                               the fp64 result to about 1e-6 (typical) .. 1e-4 (99.9 %) absolute; about 1.4x the
                               fp64 throughput for n <= SS_WARP_MAX_N.                                             */
    int shared_times;       /* 1 = every object of the catalog has the SAME time stamps in the same order (one field
                               observed together).  The fold and the sort are then done once per
                               frequency for 4 objects at a time (objects of n <= SS_GROUP_LONG_MAX_N, fp64 precision,
                               default listing options; otherwise the objects are served one by one as usual).
                               Checked on the device unless skip_validation is set: a catalog
                               whose time arrays differ is SS_ERR_INVALID_ARG.  Results equal those of
                               shared_times = 0 to rounding (same arithmetic, same order).                   */
    void *workspace;        /* device entry points: a DEVICE buffer of workspace_bytes bytes (256-byte aligned) the library
                               carves its workspace from instead of allocating; ss_workspace_bytes() is an upper bound
                               of the need.  NULL = the library allocates (and keeps the buffer for the next call).     */
    size_t workspace_bytes;
    const int64_t *offsets_host; /* device entry points: a HOST copy of `offsets`.  The batch planner needs the objects'
                               sizes on the host; without this copy the call reads `offsets` back and waits for it.    */
    int async_mode;         /* ss_periodogram_ex only.  1 = enqueue everything on opt->stream and return without waiting;
                               needs skip_validation = 1 and offsets_host (nothing is then read back).  The call is
                               completed -- status, profile counters, the hand-over overflow fallback, release of the
                               workspace -- by ss_synchronize(), or implicitly by this thread's next library call.
                               Inputs, outputs and a caller-supplied workspace must stay valid until then.               */
    unsigned int defer_capacity; /* test hook: entries of the list through which the warp-per-eval kernels hand
                               tied / undecidable evals to the generic kernel, per tile (0 = 2^20).  When it
                               overflows the call repeats itself on the CTA-per-eval kernels; results never
                               depend on it.                                                              */
} ss_options_t;

/* Fill *opt with the defaults listed above. */
void ss_default_options(ss_options_t *opt);

/*
 * DEVICE-pointer entry point (PAPER.md:88-117 over a catalog).
 *   times, mags, errs : const double[offsets[n_objects]]   device, read only
 *   offsets           : const int64_t[n_objects + 1]       device, offsets[0] == 0, non-decreasing
 *   pgram_out         : double[n_objects * n_freq] row-major device, or NULL (not materialised)
 *   best_freq_out     : double[n_objects]  device, f_min + k* * df, or NULL
 *   best_index_out    : int64_t[n_objects] device, k*, or NULL
 * Work is enqueued on the legacy default stream; the call returns after it has completed.
 */
ss_status_t ss_periodogram(const double *times, const double *mags, const double *errs,
                           const int64_t *offsets, int64_t n_objects,
                           double f_min, double f_max, int64_t n_freq, ss_mode_t mode,
                           double *pgram_out, double *best_freq_out, int64_t *best_index_out);

/* Same with options; enqueues on opt->stream and returns after that stream's work has completed -- unless
 * opt->async_mode is set (see ss_options_t), in which case it returns as soon as the work is enqueued. */
ss_status_t ss_periodogram_ex(const double *times, const double *mags, const double *errs,
                              const int64_t *offsets, int64_t n_objects,
                              double f_min, double f_max, int64_t n_freq, ss_mode_t mode,
                              double *pgram_out, double *best_freq_out, int64_t *best_index_out,
                              const ss_options_t *opt);

/*
 * HOST-pointer entry point: same operation, all array arguments are HOST pointers (pageable or
 * pinned).  The library copies the catalog to the device, tiles objects x frequencies with the batch
 * planner so the device-side periodogram tile plus workspace stays under opt->workspace_cap
 * (the batching scheme), overlaps the device->host copy of finished tiles with the
 * next tile's kernels, and returns when every output has landed in host memory.  The overlap needs
 * PAGE-LOCKED output arrays (cudaHostAlloc / cudaHostRegister): a copy into pageable memory blocks the
 * host until it is done, so the next tile's kernels are launched only afterwards -- same results, the
 * copies and the kernels then alternate instead of overlapping (bench.py's e2e leg uses pinned buffers).
 */
ss_status_t ss_periodogram_host(const double *times, const double *mags, const double *errs,
                                const int64_t *offsets, int64_t n_objects,
                                double f_min, double f_max, int64_t n_freq, ss_mode_t mode,
                                double *pgram_out, double *best_freq_out, int64_t *best_index_out,
                                const ss_options_t *opt);

/* Completes this thread's pending asynchronous ss_periodogram_ex call (opt->async_mode): waits for its stream, repeats
 * the call on the CTA-per-eval kernels if the hand-over list overflowed, releases the workspace and returns the call's
 * final status.  SS_OK when nothing is pending. */
ss_status_t ss_synchronize(void);

/* ------------------------------------------------------------------ the entry point that allocates nothing */

/* Size of the library's built-in device scratch: a file-scope `static __device__` array, so EVERY GPU that loads the
 * library holds these bytes until the process exits. */
#define SS_STATIC_SCRATCH_BYTES (32u << 20)

/*
 * The operation of ss_periodogram (Algorithm 1; 125), for callers that cannot tolerate a device
 * allocation: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  Same DEVICE-pointer
 * arguments, same kernels, default options; the workspace those kernels need (the centred copy of the catalog, object
 * records, partial-argmax rows, the hand-over list, counters) is carved from the built-in scratch array of
 * SS_STATIC_SCRATCH_BYTES instead of the pooled cudaMalloc buffer.  The call makes no cudaMalloc / cudaFree / stream or
 * event creation and calls no allocating library routine (it does use host memory of the C++ runtime).
 *
 *   offsets_host   HOST copy of offsets (n_objects + 1 values), required: the call reads no device memory from the host
 *                  except one 4-byte status flag.
 *   stream         cudaStream_t of the caller (0 = the legacy default stream); the call returns once it is complete.
 *
 * Limit: the catalog must fit the scratch -- about 24 B per point + 100 B per object + 1 MB (hand-over list of 65,536
 * entries) + the partial-argmax rows of one frequency tile (the planner tiles frequencies to fit); light curves of more
 * than SS_GROUP_MAX_N points need per-CTA staging space far beyond it.  A catalog that does not fit is rejected with
 * SS_ERR_UNSUPPORTED and a message that states the bytes needed, before anything is launched or written.
 * Sharing: every call on a device uses the SAME array; it keeps the previous call's contents (the call clears what it
 * needs zeroed), and two calls that overlap on one GPU -- from two host threads, or on two streams -- race.  Serialise them.
 * Results equal those of ss_periodogram bit for bit (same kernels, same tiling rules).
 */
ss_status_t ss_periodogram_static(const double *times, const double *mags, const double *errs,
                                  const int64_t *offsets, const int64_t *offsets_host, int64_t n_objects,
                                  double f_min, double f_max, int64_t n_freq, ss_mode_t mode,
                                  double *pgram_out, double *best_freq_out, int64_t *best_index_out, void *stream);

/* ------------------------------------------------------------------ top-k peaks */

#define SS_MAX_PEAKS 32

/*
 * The n_peaks highest PEAKS of every periodogram row.  Algorithm 1 returns only the argmax, but the
 * daily cadence of ground-based surveys aliases the true period into several comparable maxima (Fig. 1),
 * so a caller usually wants the leading candidates.  A peak is a local maximum of the row:
 *     P[k] > P[k-1]  and  P[k] >= P[k+1]
 * (a neighbour outside the grid does not disqualify; of a flat top the first index counts; NaN never qualifies).
 * Per object the peaks are ordered by falling power, equal powers by rising index; rows with fewer than n_peaks
 * peaks are padded with index -1, power NaN, frequency NaN.  peak 0 of a row is its argmax whenever the argmax is
 * unique.
 *   pgram          : const double[n_objects][row_stride], row-major, columns 0 .. n_freq-1 used (what ss_periodogram*
 *                    wrote: row_stride = n_freq, or k_count for a grid sub-range -- then pass the sub-range's own
 *                    f_min + k_begin*df as f_min and its end as f_max)
 *   peak_index_out : int64_t[n_objects][n_peaks]   column index k
 *   peak_power_out : double [n_objects][n_peaks]   P[k]                       (may be NULL)
 *   peak_freq_out  : double [n_objects][n_peaks]   f_min + k*(f_max-f_min)/n_freq   (may be NULL)
 * ss_periodogram_peaks: DEVICE pointers, work enqueued on `stream` (cudaStream_t; NULL = default stream), returns
 * after it completed.  ss_periodogram_peaks_host: HOST pointers; rows go through the device in slabs.
 * 1 <= n_peaks <= SS_MAX_PEAKS, n_freq >= 1, row_stride >= n_freq, else SS_ERR_INVALID_ARG.
 */
ss_status_t ss_periodogram_peaks(const double *pgram, int64_t n_objects, int64_t n_freq, int64_t row_stride,
                                 double f_min, double f_max, int n_peaks, int64_t *peak_index_out,
                                 double *peak_power_out, double *peak_freq_out, void *stream);
ss_status_t ss_periodogram_peaks_host(const double *pgram, int64_t n_objects, int64_t n_freq, int64_t row_stride,
                                      double f_min, double f_max, int n_peaks, int64_t *peak_index_out,
                                      double *peak_power_out, double *peak_freq_out);

/* ------------------------------------------------------------------ batch planner (host only) */

typedef struct {
    int64_t n_freq_tiles;     /* number of frequency tiles (the paper's N_b, Eq. 1)                    */
    int64_t freq_per_tile;    /* frequencies per tile (last tile may be shorter)                       */
    int64_t n_object_tiles;   /* number of object tiles                                                */
    int64_t objects_per_tile; /* objects per tile (last may be shorter)                                */
    size_t tile_bytes;        /* device bytes of one periodogram tile buffer (host entry point: x2)    */
    size_t fixed_bytes;       /* catalog copy + per-object records + scheduler state                   */
    size_t stage_bytes;       /* global staging scratch for SS_PATH_STAGE objects                      */
    size_t total_bytes;       /* what the call will allocate                                           */
} ss_plan_t;

/*
 * The plan ss_periodogram_host would use.  host_tiles != 0: output tiles are device buffers that are
 * copied back (host entry point); 0: the caller's device pgram_out is written directly.
 * Returns SS_ERR_OUT_OF_MEMORY if even a 1 x 1 tile does not fit under cap.
 */
ss_status_t ss_plan(int64_t n_points_total, int64_t max_n, int64_t n_objects, int64_t n_freq,
                    ss_mode_t mode, size_t cap_bytes, int host_tiles, int want_pgram,
                    ss_plan_t *plan_out);

/* Device bytes the library allocates for a call (planner query; = plan.total_bytes). */
size_t ss_workspace_bytes(int64_t n_points_total, int64_t max_n, int64_t n_objects,
                          int64_t n_freq, ss_mode_t mode);

/* The paper's own footprint model, for comparison and tests: bytes of its N_t*N_f layout
 * (15*N_t*N_f words) and Eq. 1's N_b = ceil(r / (beta*s)) with r from
 * PAPER.md:357/363 (FP64).  */
double ss_paper_footprint_bytes(int64_t n_t, int64_t n_f);
int64_t ss_paper_batches(int64_t n_t, int64_t n_f, ss_mode_t mode, double device_gib, double beta);

/* Path class the library picks for an object of n points (SS_PATH_WARP / GROUP / CLUSTER / STAGE; SS_PATH_BLOCK serves
 * the listing's options and whatever the other paths hand over). */
int ss_path_for_n(int64_t n, ss_mode_t mode);

/* ------------------------------------------------------------------ diagnostics */

/* Smoothed values of ONE (object, frequency) eval, in phase order, plus the permutation
 * (device pointers; smo_out double[n], perm_out int32_t[n], either may be NULL).  Test hook. */
ss_status_t ss_debug_eval(const double *times, const double *mags, const double *errs, int64_t n,
                          double freq, ss_mode_t mode, const ss_options_t *opt,
                          double *smo_out, int32_t *perm_out, double *p_out);

/* Microbenchmarks used for the roofline denominators: sustained fp64 FMA
 * rate (FLOP/s, 2 per DFMA) and shared-memory read bandwidth (B/s) of this device. */
ss_status_t ss_microbench(double *fp64_flops_out, double *smem_bytes_per_s_out, void *stream);

/* Kernel launches issued by this thread's most recent ss_periodogram* call. */
int64_t ss_last_launch_count(void);

/* With opt->profile = 1: total device time (ms, CUDA events on the launching stream) and number of
 * the eval-kernel launches (warp/block/stage kernels) of this thread's most recent call. */
double ss_last_kernel_ms(void);
int64_t ss_last_kernel_count(void);

/* The library keeps the device buffers, events and the copy stream of a thread's most recent calls for
 * reuse by its next call (a call in steady state makes no cudaMalloc/cudaFree; at most 4 buffers per thread:
 * workspace, and for the host entry point the catalog copy and two output tiles).  This frees them. */
void ss_release_workspace(void);

const char *ss_last_error(void); /* thread-local, never NULL */
int ss_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SS_PERIODOGRAM_H */
