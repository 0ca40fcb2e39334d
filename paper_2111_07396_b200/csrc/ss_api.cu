// ss_api.cu -- C-ABI entry points, host driver (Algorithm 1, restructured so that
// nothing is materialised at N_t*N_f), prep / argmax / fill kernels and the microbenchmarks.
#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <memory>
#include <string>
#include <mutex>
#include <vector>

#include "../../include/ss_periodogram.h"
#include "ss_common.cuh"
#include "ss_launch.h"
#include "ss_planner.h"

namespace ss {

static thread_local std::string g_err = "";
static thread_local int64_t g_launches = 0;
static thread_local double g_kernel_ms = 0.0;
static thread_local int64_t g_kernel_count = 0;

static ss_status_t fail(ss_status_t st, const char* fmt, ...)
{
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    g_err = buf;
    return st;
}

#define SS_CUDA(call)                                                                        \
    do {                                                                                     \
        cudaError_t e_ = (call);                                                             \
        if (e_ != cudaSuccess)                                                               \
            return fail(e_ == cudaErrorMemoryAllocation ? SS_ERR_OUT_OF_MEMORY : SS_ERR_CUDA, \
                        "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__); \
    } while (0)

// ------------------------------------------------------------------------------------------------
// Per-thread device resources kept between calls: a call in steady state makes no cudaMalloc / cudaFree /
// event or stream creation (each of those enters the driver's resource manager, where it can queue behind
// other clients of the GPU -- measured: up to 0.4 s per call while nvidia-smi polls the device).  The pool
// holds at most POOL_SLOTS buffers; ss_release_workspace() frees everything.
// ------------------------------------------------------------------------------------------------
constexpr int POOL_SLOTS = 4;
struct DevicePool {
    struct Buf { char* p = nullptr; size_t bytes = 0; int dev = -1; };
    Buf bufs[POOL_SLOTS];
    std::vector<cudaEvent_t> timing_events, plain_events;
    cudaStream_t copy_stream = nullptr;
    int copy_stream_dev = -1;
    int event_dev = -1;

    // smallest cached buffer of this device that is large enough, else a fresh allocation
    cudaError_t acquire(size_t bytes, char** out)
    {
        int dev = 0;
        cudaError_t e = cudaGetDevice(&dev);
        if (e != cudaSuccess) return e;
        int best = -1;
        for (int i = 0; i < POOL_SLOTS; i++)
            if (bufs[i].p && bufs[i].dev == dev && bufs[i].bytes >= bytes && (best < 0 || bufs[i].bytes < bufs[best].bytes)) best = i;
        if (best >= 0 && bufs[best].bytes <= 2 * bytes + (64u << 20)) {      // do not pin a huge buffer on a small request
            *out = bufs[best].p;
            bufs[best] = Buf{};
            return cudaSuccess;
        }
        e = cudaMalloc((void**)out, bytes);
        if (e == cudaErrorMemoryAllocation) {      // make room: drop the cache and try once more
            release_all();
            cudaGetLastError();
            e = cudaMalloc((void**)out, bytes);
        }
        return e;
    }
    void release(char* p, size_t bytes)
    {
        if (!p) return;
        int dev = 0;
        cudaGetDevice(&dev);
        int slot = -1;
        for (int i = 0; i < POOL_SLOTS; i++) if (!bufs[i].p) { slot = i; break; }
        if (slot < 0) {                            // full: evict the smallest
            slot = 0;
            for (int i = 1; i < POOL_SLOTS; i++) if (bufs[i].bytes < bufs[slot].bytes) slot = i;
            if (bufs[slot].bytes >= bytes) { cudaFree(p); return; }
            cudaFree(bufs[slot].p);
        }
        bufs[slot] = Buf{p, bytes, dev};
    }
    cudaError_t event(bool timing, cudaEvent_t* out)
    {
        // events belong to the device they were created on: a thread that switched devices starts a fresh cache
        int dev = 0;
        cudaGetDevice(&dev);
        if (dev != event_dev) {
            for (auto e : timing_events) cudaEventDestroy(e);
            for (auto e : plain_events) cudaEventDestroy(e);
            timing_events.clear(); plain_events.clear();
            event_dev = dev;
        }
        auto& v = timing ? timing_events : plain_events;
        if (!v.empty()) { *out = v.back(); v.pop_back(); return cudaSuccess; }
        return timing ? cudaEventCreate(out) : cudaEventCreateWithFlags(out, cudaEventDisableTiming);
    }
    void event_back(bool timing, cudaEvent_t e) { if (e) (timing ? timing_events : plain_events).push_back(e); }
    cudaError_t stream(cudaStream_t* out)
    {
        int dev = 0;
        cudaGetDevice(&dev);
        if (copy_stream && copy_stream_dev != dev) { cudaStreamDestroy(copy_stream); copy_stream = nullptr; }
        if (!copy_stream) {
            cudaError_t e = cudaStreamCreateWithFlags(&copy_stream, cudaStreamNonBlocking);
            if (e != cudaSuccess) return e;
            copy_stream_dev = dev;
        }
        *out = copy_stream;
        return cudaSuccess;
    }
    void release_all()
    {
        for (auto& b : bufs) { if (b.p) cudaFree(b.p); b = Buf{}; }
        for (auto e : timing_events) cudaEventDestroy(e);
        for (auto e : plain_events) cudaEventDestroy(e);
        timing_events.clear(); plain_events.clear();
        if (copy_stream) { cudaStreamDestroy(copy_stream); copy_stream = nullptr; }
    }
};
static thread_local DevicePool g_pool;
static_assert(sizeof(ObjRec) == OBJREC_BYTES, "planner's record size");

// ------------------------------------------------------------------------------------------------
// P0 prep: tt = t - min t, w = e^-2, ybar_w, chi0; yc = y - ybar_w.
// One CTA per object.  Also validates: finite t, y, e and e > 0 (flag[0] |= 1 otherwise).
// ------------------------------------------------------------------------------------------------
constexpr int PREP_T = 256;

__device__ __forceinline__ double prep_block_sum(double v, double* red)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
    __syncthreads();
    if (lane == 0) red[warp] = v;
    __syncthreads();
    double s = 0.0;
    for (int q = 0; q < PREP_T / 32; q++) s += red[q];
    return s;
}

// raw_off[ri]: the object's first element in the caller's arrays; recs[ri].off: its first element in tt / yc / w
// (every object starts at an even element there: 16-byte aligned for the bulk copies of the group kernel).
__global__ void __launch_bounds__(PREP_T) prep_kernel(const double* __restrict__ times,
                                                      const double* __restrict__ mags,
                                                      const double* __restrict__ errs, ObjRec* recs,
                                                      const int64_t* __restrict__ raw_off,
                                                      int n_recs, double* tt, double* yc, double* w,
                                                      int* flag)
{
    __shared__ double red[PREP_T / 32];
    const int ri = blockIdx.x;
    if (ri >= n_recs) return;
    const int64_t off = raw_off[ri], poff = recs[ri].off;
    const int n = recs[ri].n;
    const int tid = threadIdx.x;
    double tmin = INFINITY;
    int bad = 0;
    for (int j = tid; j < n; j += PREP_T) {
        double t = times[off + j], y = mags[off + j], e = errs[off + j];
        if (!isfinite(t) || !isfinite(y) || !isfinite(e) || !(e > 0.0)) bad = 1;
        tmin = fmin(tmin, t);
    }
    if (bad) atomicOr(flag, 1);
    // duplicated time stamps tie at every frequency: the warp path hands such an object over whole (ObjRec::dup)
    if (n <= SS_WARP_MAX_N) {
        int dup = 0;
        for (int j = tid; j < n; j += PREP_T) {
            const double t = times[off + j];
            for (int i = 0; i < j; i++) dup |= (times[off + i] == t);
        }
        dup = __syncthreads_or(dup);
        if (tid == 0) recs[ri].dup = dup ? 1 : 0;
    }
    // block min
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) tmin = fmin(tmin, __shfl_xor_sync(0xffffffffu, tmin, d));
    __syncthreads();
    if ((tid & 31) == 0) red[tid >> 5] = tmin;
    __syncthreads();
    tmin = red[0];
    for (int q = 1; q < PREP_T / 32; q++) tmin = fmin(tmin, red[q]);
    double sw = 0.0, swy = 0.0;
    // centre on the first magnitude before summing so the weighted mean keeps full precision
    const double y0 = mags[off];
    for (int j = tid; j < n; j += PREP_T) {
        double e = errs[off + j];
        double wj = 1.0 / (e * e);
        w[poff + j] = wj;
        tt[poff + j] = times[off + j] - tmin;
        sw += wj;
        swy += wj * (mags[off + j] - y0);
    }
    sw = prep_block_sum(sw, red);
    swy = prep_block_sum(swy, red);
    const double ybar = y0 + swy / sw;
    double c0 = 0.0;
    for (int j = tid; j < n; j += PREP_T) {
        double d = mags[off + j] - ybar;
        yc[poff + j] = d;
        c0 += w[poff + j] * d * d;
    }
    c0 = prep_block_sum(c0, red);
    if (tid == 0) {
        if (n & 1) { tt[poff + n] = 0.0; yc[poff + n] = 0.0; w[poff + n] = 0.0; }      // the padding element
        recs[ri].chi0 = c0;
        recs[ri].ybar = ybar;
    }
}

// shared_times = 1: every object must carry the time stamps of the first one (flag |= 2 otherwise)
__global__ void shared_times_check_kernel(const double* __restrict__ times, const ObjRec* recs,
                                          const int64_t* __restrict__ raw_off, int n_recs, int* flag)
{
    const int ri = blockIdx.x + 1;
    if (ri >= n_recs) return;
    const int n = recs[ri].n;
    const int64_t a = raw_off[0], b = raw_off[ri];
    int bad = recs[0].n != n;
    for (int j = threadIdx.x; j < n && !bad; j += blockDim.x) bad |= times[a + j] != times[b + j];
    if (bad) atomicOr(flag, 2);
}

// Fold one tile's partial maxima into the running best of each object (O8: first maximum wins).
__global__ void fold_best_kernel(const ObjRec* recs, const int32_t* list, int n_list, int chunks,
                                 int chunks_total, int chunk_base, const double* part_val,
                                 const int64_t* part_idx, double* best_val, int64_t* best_idx)
{
    const int gw = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (gw >= n_list) return;
    const int ri = list[gw];
    double bv = -INFINITY;
    int64_t bk = INT64_MAX;
    for (int c = lane; c < chunks; c += 32) {
        int64_t slot = (int64_t)ri * chunks_total + chunk_base + c;
        double v = part_val[slot];
        int64_t k = part_idx[slot];
        if (v > bv || (v == bv && k < bk)) { bv = v; bk = k; }
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        double ov = __shfl_xor_sync(0xffffffffu, bv, d);
        int64_t ok = __shfl_xor_sync(0xffffffffu, bk, d);
        if (ov > bv || (ov == bv && ok < bk)) { bv = ov; bk = ok; }
    }
    if (lane == 0) {
        const int64_t o = recs[ri].obj;
        double cv = best_val[o];
        int64_t ck = best_idx[o];
        if (ck < 0 || bv > cv || (bv == cv && bk < ck)) { best_val[o] = bv; best_idx[o] = bk; }
    }
}

__global__ void init_best_kernel(int64_t n, double* best_val, int64_t* best_idx)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) { best_val[i] = -INFINITY; best_idx[i] = -1; }
}

// best_index = k*, best_freq = f_min + k* df; objects that were never evaluated
// (n < 5) keep index -1 and get NaN.
__global__ void finish_kernel(int64_t n, const int64_t* best_idx, double f_min, double df,
                              double* best_freq_out, int64_t* best_index_out)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int64_t k = best_idx[i];
    if (best_index_out) best_index_out[i] = k;
    if (best_freq_out) best_freq_out[i] = k >= 0 ? freq_of(f_min, df, k) : nan("");
}

// NaN rows for degenerate objects (n < 5).
__global__ void nan_rows_kernel(const int64_t* rows, int n_rows, int64_t row0, int64_t width,
                                int64_t stride, double* pgram)
{
    const int r = blockIdx.y;
    if (r >= n_rows) return;
    int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c < width) pgram[(rows[r] - row0) * stride + c] = nan("");
}

// ------------------------------------------------------------------------------------------------
// Microbenchmarks for the roofline denominators.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) fp64_peak_kernel(double* out, int iters)
{
    double a[8];
    const double m = 1.0000001, c = 1e-9;
#pragma unroll
    for (int i = 0; i < 8; i++) a[i] = threadIdx.x * 1e-3 + i;
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int i = 0; i < 8; i++) a[i] = fma(a[i], m, c);
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 8; i++) s += a[i];
    if (s == 12345.678) out[0] = s;
}

__global__ void __launch_bounds__(256) smem_peak_kernel(double* out, int iters)
{
    __shared__ double buf[4096];
    for (int i = threadIdx.x; i < 4096; i += 256) buf[i] = i;
    __syncthreads();
    double s = 0;
    int idx = threadIdx.x;
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int u = 0; u < 8; u++) {
            s += buf[(idx + u * 256) & 4095];
        }
        idx = (idx + 37) & 4095;
    }
    if (s == 12345.678) out[0] = s;
}

// ------------------------------------------------------------------------------------------------
// Engine: device state of one call.
// ------------------------------------------------------------------------------------------------
struct ClassList {
    int path;               // SS_PATH_*
    int variant;            // path-specific sub-class (warp: points per lane; block: smem tier)
    std::vector<int32_t> recs;   // record indices, longest first
    int64_t list_off = 0;   // offset into the device list array
    int max_n = 0;
};

struct Engine {
    cudaStream_t stream = nullptr;
    ss_options_t opt{};
    int mode = 0;
    int64_t n_objects = 0, n_freq = 0, total = 0;
    int64_t k_lo = 0, k_n = 0;         // the sub-range of the grid this call evaluates (opt.k_begin / k_count)
    double f_min = 0, df = 0;
    std::vector<int64_t> off;
    std::vector<ObjRec> recs;          // objects with n >= 5
    std::vector<int64_t> degenerate;   // object indices with n < 5
    std::vector<int64_t> raw_off;      // per record: first element in the caller's arrays
    int64_t padded_total = 0;          // elements of tt / yc / w (every object padded to an even length)
    int64_t* d_raw_off = nullptr;
    int max_n = 0;
    // device workspace
    char* ws = nullptr;
    size_t ws_bytes = 0;
    bool ws_owned = true;              // false: the caller's buffer (opt.workspace)
    double *tt = nullptr, *yc = nullptr, *w = nullptr;
    ObjRec* d_recs = nullptr;
    int32_t* d_list = nullptr;
    int64_t* d_degen = nullptr;
    double* best_val = nullptr;
    int64_t* best_idx = nullptr;
    double* part_val = nullptr;
    int64_t* part_idx = nullptr;
    unsigned int* counters = nullptr;
    int* flag = nullptr;
    double* stage = nullptr;
    unsigned long long* defer_entries = nullptr;   // warp path -> generic kernel hand-over
    double* defer_val = nullptr;
    unsigned int* defer_count = nullptr;
    unsigned long long *dmax = nullptr, *dmin = nullptr;
    unsigned int defer_capacity = DEFER_CAPACITY;
    char* extra = nullptr;            // caller-requested extra bytes (host entry point buffers)
    int64_t stage_stride = 0;
    int n_counters = 0, next_counter = 0;
    ss_plan_t plan{};
    // per object tile: class lists
    std::vector<std::vector<ClassList>> tiles;
    int sm_count = 148;
    std::vector<std::pair<cudaEvent_t, cudaEvent_t>> prof;   // opt.profile: events around eval kernels

    ~Engine()
    {
        // pooled buffers must be idle when they go back (already true unless the call is failing)
        if (ws) cudaStreamSynchronize(stream);
        for (auto& e : prof) { g_pool.event_back(true, e.first); g_pool.event_back(true, e.second); }
        if (ws_owned) g_pool.release(ws, ws_bytes);
    }
    // After the stream is synchronised: did the deferred list overflow?
    bool defer_overflowed()
    {
        unsigned int h[2] = {0, 0};
        if (!defer_count) return false;
        if (cudaMemcpy(h, defer_count, 8, cudaMemcpyDeviceToHost) != cudaSuccess) return false;
        return h[1] != 0;
    }
    // Sum the profiled kernel times (call after the stream has been synchronised).
    void collect_profile()
    {
        g_kernel_ms = 0.0; g_kernel_count = (int64_t)prof.size();
        for (auto& e : prof) { float ms = 0; if (cudaEventElapsedTime(&ms, e.first, e.second) == cudaSuccess) g_kernel_ms += ms; }
    }

    ss_status_t setup(const double* times, const double* mags, const double* errs,
                      const int64_t* offsets_host, int64_t n_obj, double fmin, double fmax,
                      int64_t nfreq, int md, const ss_options_t& o, bool host_tiles, bool want_pgram,
                      size_t extra_bytes);
    ss_status_t run_tile(int obj_tile, int64_t k_begin, int64_t k_end, int freq_tile_index,
                         double* pgram, int64_t row_stride, int64_t row0, int64_t k0);
    ss_status_t finish(double* best_freq_out, int64_t* best_index_out);
};

static ss_status_t validate_scalars(int64_t n_objects, double f_min, double f_max, int64_t n_freq,
                                    int mode, const ss_options_t& o)
{
    if (n_objects < 0) return fail(SS_ERR_INVALID_ARG, "n_objects < 0");
    if (n_freq < 1) return fail(SS_ERR_INVALID_ARG, "n_freq < 1");
    if (!(f_min > 0.0) || !std::isfinite(f_min)) return fail(SS_ERR_INVALID_ARG, "f_min must be finite and > 0");
    if (!(f_max > f_min) || !std::isfinite(f_max)) return fail(SS_ERR_INVALID_ARG, "f_max must be finite and > f_min");
    if (mode != SS_MODE_CROSS_VALIDATION && mode != SS_MODE_GENERALIZED_VALIDATION)
        return fail(SS_ERR_INVALID_ARG, "unknown mode %d", mode);
    if (!(o.span >= 0.0) || !(o.span <= 1.0)) return fail(SS_ERR_INVALID_ARG, "span must be 0 (variable) or in (0, 1]");
    if (o.iper != 1 && o.iper != 2) return fail(SS_ERR_INVALID_ARG, "iper = %d (1 = non-periodic, 2 = periodic)", o.iper);
    if (!std::isfinite(o.alpha)) return fail(SS_ERR_INVALID_ARG, "alpha is not finite");
    if (o.precision != SS_PRECISION_F64 && o.precision != SS_PRECISION_MIXED)
        return fail(SS_ERR_INVALID_ARG, "precision = %d (0 = fp64, 1 = mixed)", o.precision);
    if (o.k_begin < 0 || o.k_count < 0 || o.k_begin >= n_freq || o.k_begin + o.k_count > n_freq)
        return fail(SS_ERR_INVALID_ARG, "k_begin/k_count outside the grid");
    return SS_OK;
}

// SM count of the current device; the B200's when no device is visible (planner queries on a CPU-only box)
static int device_sm_count()
{
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0) {
        cudaGetLastError();
        return DEFAULT_SM_COUNT;
    }
    return sms;
}

static bool has_listing_options(const ss_options_t& o) { return o.iper == 2 || o.span > 0.0; }

static size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }

ss_status_t Engine::setup(const double* times, const double* mags, const double* errs,
                          const int64_t* offsets_host, int64_t n_obj, double fmin, double fmax,
                          int64_t nfreq, int md, const ss_options_t& o, bool host_tiles,
                          bool want_pgram, size_t extra_bytes)
{
    opt = o;
    if (o.defer_capacity > 0) defer_capacity = o.defer_capacity;
    stream = (cudaStream_t)o.stream;
    mode = md;
    n_objects = n_obj;
    n_freq = nfreq;
    k_lo = o.k_begin;
    k_n = o.k_count > 0 ? o.k_count : nfreq - o.k_begin;
    f_min = fmin;
    df = (fmax - fmin) / (double)nfreq;
    int dev = 0;
    SS_CUDA(cudaGetDevice(&dev));
    SS_CUDA(cudaDeviceGetAttribute(&sm_count, cudaDevAttrMultiProcessorCount, dev));

    off.assign(offsets_host, offsets_host + n_obj + 1);
    if (n_obj > 0 && off[0] != 0) return fail(SS_ERR_INVALID_ARG, "offsets[0] != 0");
    for (int64_t i = 0; i < n_obj; i++)
        if (off[i + 1] < off[i]) return fail(SS_ERR_INVALID_ARG, "offsets not non-decreasing at %lld", (long long)i);
    total = n_obj > 0 ? off[n_obj] : 0;
    for (int64_t i = 0; i < n_obj; i++) {
        int64_t n = off[i + 1] - off[i];
        if (n > (int64_t)1 << 24) return fail(SS_ERR_UNSUPPORTED, "object %lld has %lld points (limit 2^24)", (long long)i, (long long)n);
        if (n < MIN_POINTS) { degenerate.push_back(i); continue; }
        ObjRec r{};
        r.off = padded_total; r.obj = i; r.n = (int32_t)n;
        raw_off.push_back(off[i]);
        padded_total += (n + 1) & ~(int64_t)1;
        r.ibw[0] = half_width(n, SPAN0); r.ibw[1] = half_width(n, SPAN1); r.ibw[2] = half_width(n, SPAN2);
        r.q1 = (int32_t)(n / 4 - 1); r.q3 = 3 * (r.q1 + 1) - 1;
        r.ibw_fixed = o.span > 0.0 ? half_width(n, o.span) : 0;
        recs.push_back(r);
        max_n = std::max(max_n, (int)n);
    }

    // ---- plan (P6)
    size_t cap = o.workspace_cap;
    if (cap == 0) {
        size_t fr = 0, tot = 0;
        SS_CUDA(cudaMemGetInfo(&fr, &tot));
        cap = (size_t)(0.75 * (double)fr);   // the paper's beta
    }
    PlanInput pin{total, max_n, n_obj, k_n, md, cap, host_tiles ? 1 : 0, want_pgram ? 1 : 0, o.freq_tile, sm_count, defer_capacity};
    ss_status_t st = make_plan(pin, &plan);
    if (st != SS_OK) return fail(st, "workspace cap %zu B too small for the smallest tile", cap);

    // ---- class lists per object tile
    const int n_ot = (int)std::max<int64_t>(plan.n_object_tiles, 1);
    tiles.assign(n_ot, {});
    std::vector<int32_t> all_lists;
    for (int t = 0; t < n_ot; t++) {
        const int64_t o0 = (int64_t)t * plan.objects_per_tile, o1 = std::min(n_obj, o0 + plan.objects_per_tile);
        std::vector<ClassList> cls;
        auto find = [&](int path, int variant) -> ClassList& {
            for (auto& c : cls) if (c.path == path && c.variant == variant) return c;
            cls.push_back(ClassList{path, variant, {}, 0, 0});
            return cls.back();
        };
        for (size_t ri = 0; ri < recs.size(); ri++) {
            const ObjRec& r = recs[ri];
            if (r.obj < o0 || r.obj >= o1) continue;
            int path = o.force_path != SS_PATH_AUTO ? o.force_path : path_for_n(r.n, md);
            // periodic windows and the fixed span: the warp and group paths have their own kernels for them, longer
            // light curves go to the generic CTA-per-eval code
            if (path == SS_PATH_WARP && (r.n > SS_WARP_MAX_N || !WARP_IMPLEMENTED)) path = SS_PATH_GROUP;
            // a fixed span narrower than the tweeter's: a window sum is then < 1/20 of the prefixes it is the difference
            // of, and a near-singular window (7 points inside a seasonal gap's edge) misses the 1e-9 bar by prefix
            // differences at n > 256 (measured 1.03e-9); the CTA-per-eval kernels sum such windows directly
            if (path == SS_PATH_GROUP && o.span > 0.0 && o.span < SPAN0) path = SS_PATH_BLOCK;
            if (path == SS_PATH_GROUP && r.n > SS_GROUP_LONG_MAX_N) path = SS_PATH_CLUSTER;
            if (path == SS_PATH_CLUSTER && has_listing_options(o)) path = SS_PATH_STAGE;
            if (path == SS_PATH_CLUSTER && (r.n > SS_CLUSTER_MAX_N || r.n < 2 * 512)) path = SS_PATH_STAGE;
            if (path == SS_PATH_BLOCK && r.n > BLOCK_MAX_N) path = SS_PATH_STAGE;
            int variant = 0;
            if (path == SS_PATH_WARP)
                variant = has_listing_options(o) ? WARP_VARIANT_OPT + std::max(2, (r.n + 31) / 32)
                                                 : warp_variant_for_n(r.n) + (o.precision == SS_PRECISION_MIXED ? WARP_VARIANT_F32 : 0);
            else if (path == SS_PATH_GROUP)
                variant = group_variant_for_n(r.n) + (has_listing_options(o) ? GROUP_VARIANT_OPT
                                                      : o.precision == SS_PRECISION_MIXED ? GROUP_VARIANT_F32 : 0);
            else if (path == SS_PATH_CLUSTER) variant = cluster_variant_for_n(r.n);
            // CTA size by n (profiles/r1g_crossover.md): 128 threads up to 512 points, 256 up to 1,020, 512 beyond
            else if (path == SS_PATH_BLOCK) variant = r.n <= 512 ? 3 : (r.n <= 1020 ? 1 : 2);
            ClassList& c = find(path, variant);
            c.recs.push_back((int32_t)ri);
            c.max_n = std::max(c.max_n, (int)r.n);
        }
        for (auto& c : cls) {
            std::stable_sort(c.recs.begin(), c.recs.end(),
                             [&](int32_t a, int32_t b) { return recs[a].n > recs[b].n; });
            c.list_off = (int64_t)all_lists.size();
            all_lists.insert(all_lists.end(), c.recs.begin(), c.recs.end());
        }
        tiles[t] = std::move(cls);
    }

    // ---- workspace: one buffer, carved by the planner's layout function with this catalog's actual counts
    const bool need_stage = max_n > BLOCK_MAX_N || o.force_path == SS_PATH_STAGE;
    const int64_t cpo = chunks_per_object(plan.objects_per_tile, plan.freq_per_tile);
    WsCounts wc;
    wc.padded_points = padded_total; wc.n_recs = (int64_t)recs.size(); wc.n_list = (int64_t)all_lists.size();
    wc.n_degenerate = (int64_t)degenerate.size(); wc.n_objects = n_obj;
    wc.partial_slots = (int64_t)std::max<size_t>(recs.size(), 1) * cpo;
    wc.max_n = max_n; wc.stage = need_stage ? 1 : 0; wc.sm_count = sm_count; wc.defer_capacity = defer_capacity;
    const WsLayout L = ws_layout(wc);
    stage_stride = L.stage_stride;
    n_counters = WS_COUNTERS;
    ws_bytes = L.bytes + ws_align(extra_bytes);
    if (ws_bytes > cap)
        return fail(SS_ERR_OUT_OF_MEMORY, "workspace %zu B exceeds the cap %zu B", ws_bytes, cap);
    if (o.workspace) {
        // caller-supplied device workspace (ss_workspace_bytes() is an upper bound of the need)
        if (o.workspace_bytes < ws_bytes)
            return fail(SS_ERR_OUT_OF_MEMORY, "caller workspace of %zu B is smaller than the %zu B this call needs", o.workspace_bytes, ws_bytes);
        if (((uintptr_t)o.workspace & 255) != 0) return fail(SS_ERR_INVALID_ARG, "workspace must be 256-byte aligned");
        ws = (char*)o.workspace;
        ws_owned = false;
    } else {
        SS_CUDA(g_pool.acquire(ws_bytes, &ws));
    }
    tt = (double*)(ws + L.tt); yc = (double*)(ws + L.yc); w = (double*)(ws + L.w);
    d_raw_off = (int64_t*)(ws + L.raw);
    d_recs = (ObjRec*)(ws + L.recs); d_list = (int32_t*)(ws + L.list); d_degen = (int64_t*)(ws + L.degen);
    best_val = (double*)(ws + L.best_val); best_idx = (int64_t*)(ws + L.best_idx);
    part_val = (double*)(ws + L.part_val); part_idx = (int64_t*)(ws + L.part_idx);
    counters = (unsigned int*)(ws + L.counters); flag = (int*)(ws + L.flag);
    stage = need_stage ? (double*)(ws + L.stage) : nullptr;
    defer_entries = (unsigned long long*)(ws + L.defer_entries); defer_val = (double*)(ws + L.defer_val);
    defer_count = (unsigned int*)(ws + L.defer_count);
    dmax = (unsigned long long*)(ws + L.dmax); dmin = (unsigned long long*)(ws + L.dmin);
    extra = ws + L.bytes;

    if (!recs.empty()) SS_CUDA(cudaMemcpyAsync(d_recs, recs.data(), sizeof(ObjRec) * recs.size(), cudaMemcpyHostToDevice, stream));
    if (!recs.empty()) SS_CUDA(cudaMemcpyAsync(d_raw_off, raw_off.data(), 8 * raw_off.size(), cudaMemcpyHostToDevice, stream));
    if (!all_lists.empty()) SS_CUDA(cudaMemcpyAsync(d_list, all_lists.data(), 4 * all_lists.size(), cudaMemcpyHostToDevice, stream));
    if (!degenerate.empty()) SS_CUDA(cudaMemcpyAsync(d_degen, degenerate.data(), 8 * degenerate.size(), cudaMemcpyHostToDevice, stream));
    SS_CUDA(cudaMemsetAsync(counters, 0, 4 * (size_t)n_counters, stream));
    SS_CUDA(cudaMemsetAsync(flag, 0, 64, stream));
    SS_CUDA(cudaMemsetAsync(defer_count, 0, 64, stream));
    if (n_obj > 0) {
        init_best_kernel<<<(unsigned)((n_obj + 255) / 256), 256, 0, stream>>>(n_obj, best_val, best_idx);
        g_launches++;
    }
    if (!recs.empty()) {
        prep_kernel<<<(unsigned)recs.size(), PREP_T, 0, stream>>>(times, mags, errs, d_recs, d_raw_off, (int)recs.size(), tt, yc, w, flag);
        g_launches++;
        SS_CUDA(cudaGetLastError());
    }
    if (o.shared_times && !o.skip_validation && recs.size() > 1) {
        if (recs.size() != (size_t)n_obj) return fail(SS_ERR_INVALID_ARG, "shared_times: every object needs the same number of points");
        shared_times_check_kernel<<<(unsigned)recs.size() - 1, 256, 0, stream>>>(times, d_recs, d_raw_off, (int)recs.size(), flag);
        g_launches++;
    }
    if (!o.skip_validation) {
        int h_flag = 0;
        SS_CUDA(cudaMemcpyAsync(&h_flag, flag, sizeof(int), cudaMemcpyDeviceToHost, stream));
        SS_CUDA(cudaStreamSynchronize(stream));
        if (h_flag & 2) return fail(SS_ERR_INVALID_ARG, "shared_times is set but the objects' time stamps differ");
        if (h_flag) return fail(SS_ERR_INVALID_ARG, "non-finite time/magnitude/error or error <= 0 in the catalog");
    }
    return SS_OK;
}

ss_status_t Engine::run_tile(int obj_tile, int64_t k_begin, int64_t k_end, int freq_tile_index,
                             double* pgram, int64_t row_stride, int64_t row0, int64_t k0)
{
    (void)freq_tile_index;
    if (tiles.empty()) return SS_OK;
    const int64_t nk = k_end - k_begin;
    const int64_t o0 = (int64_t)obj_tile * plan.objects_per_tile, o1 = std::min(n_objects, o0 + plan.objects_per_tile);
    const int64_t cpo_cap = chunks_per_object(plan.objects_per_tile, plan.freq_per_tile);
    for (ClassList& c : tiles[obj_tile]) {
        if (c.recs.empty()) continue;
        EvalParams p{};
        p.tt = tt; p.yc = yc; p.w = w; p.recs = d_recs;
        p.list = d_list + c.list_off; p.n_list = (int32_t)c.recs.size();
        p.f_min = f_min; p.df = df; p.k_begin = k_begin; p.k_end = k_end;
        int64_t cpo = std::min<int64_t>(cpo_cap, nk);
        int64_t chunk = (nk + cpo - 1) / cpo;
        if (c.path == SS_PATH_WARP) chunk = (chunk + WARPS_PER_CTA - 1) / WARPS_PER_CTA * WARPS_PER_CTA;
        // a cluster sets up tensor memory and its window tables per work item: up to 64 evals each while that still
        // leaves a few hundred items
        if (c.path == SS_PATH_CLUSTER) {
            const int64_t want = std::max<int64_t>(1, std::min<int64_t>(64, nk * (int64_t)c.recs.size() / 256));
            if (chunk < want) chunk = want;
        }
        cpo = (nk + chunk - 1) / chunk;
        p.chunk = (int32_t)chunk; p.chunks_per_obj = (int32_t)cpo;
        p.chunks_total = (int32_t)cpo_cap; p.chunk_base = 0;
        p.alpha = opt.alpha; p.mode = mode; p.iper = opt.iper; p.span = opt.span;
        p.pgram = pgram; p.pgram_row_stride = row_stride; p.pgram_k0 = k0; p.pgram_row0 = row0;
        p.part_val = part_val; p.part_idx = part_idx;
        p.counter = counters + (next_counter % n_counters);
        p.stage = stage; p.stage_stride = stage_stride;
        p.defer_entries = defer_entries; p.defer_count = defer_count; p.defer_capacity = defer_capacity;
        // one fold + sort per group of objects (fp64 kernels with default options)
        const bool shared = opt.shared_times && ((c.path == SS_PATH_WARP && c.variant < WARP_VARIANT_F32) ||
                                                 (c.path == SS_PATH_GROUP && c.variant < GROUP_VARIANT_F32));
        const int64_t n_items = (shared ? ((int64_t)p.n_list + SHARED_TIMES_M - 1) / SHARED_TIMES_M : (int64_t)p.n_list) * cpo;
        if (n_items > 0x7fffffffLL) return fail(SS_ERR_UNSUPPORTED, "too many work items in one tile");
        cudaEvent_t ev0 = nullptr, ev1 = nullptr;
        if (opt.profile) {
            SS_CUDA(g_pool.event(true, &ev0));
            SS_CUDA(g_pool.event(true, &ev1));
            prof.emplace_back(ev0, ev1);
        }
        const bool hands_over = c.path == SS_PATH_WARP || c.path == SS_PATH_GROUP || c.path == SS_PATH_CLUSTER;   // no work counter, hand-over list
        if (!hands_over) {
            SS_CUDA(cudaMemsetAsync(p.counter, 0, 4, stream));
            next_counter++;
        }
        if (ev0) SS_CUDA(cudaEventRecord(ev0, stream));
        if (c.path == SS_PATH_WARP) {
            ss_status_t st = c.variant >= WARP_VARIANT_OPT
                                 ? launch_warp_opt_kernel(p, c.variant - WARP_VARIANT_OPT, opt.span > 0.0 ? 2 : mode, n_items, stream)
                                 : shared ? launch_warp_shared_kernel(p, c.variant, n_items, stream)
                                          : launch_warp_kernel(p, c.variant, n_items, stream);
            if (st != SS_OK) return fail(st, "warp kernel launch failed: %s", cudaGetErrorString(cudaGetLastError()));
        } else if (c.path == SS_PATH_CLUSTER) {
            ss_status_t st = launch_cluster_kernel(p, c.variant, n_items, stream);
            if (st != SS_OK) return fail(st, "cluster kernel launch failed: %s", cudaGetErrorString(cudaGetLastError()));
        } else if (c.path == SS_PATH_GROUP) {
            ss_status_t st = c.variant >= GROUP_VARIANT_OPT
                                 ? launch_group_opt_kernel(p, c.variant - GROUP_VARIANT_OPT, opt.span > 0.0 ? 2 : mode, n_items, stream)
                                 : shared ? launch_group_shared_kernel(p, c.variant, n_items, stream)
                                          : launch_group_kernel(p, c.variant, n_items, stream);
            if (st != SS_OK) return fail(st, "group kernel launch failed: %s", cudaGetErrorString(cudaGetLastError()));
        } else {
            const int threads = c.path == SS_PATH_STAGE ? 512 : (c.variant == 2 ? 512 : (c.variant == 3 ? 128 : 256));
            ss_status_t st = launch_block_kernel(p, c.path, threads, c.max_n, has_listing_options(opt), n_items, sm_count, stream);
            if (st != SS_OK) return fail(st, "CTA kernel launch failed: %s", cudaGetErrorString(cudaGetLastError()));
        }
        if (ev1) SS_CUDA(cudaEventRecord(ev1, stream));
        g_launches++;
        if (hands_over) {
            // what the warp / group path handed over (tied / misordered phases, leave-one-out denominator <= 0, objects
            // with duplicated time stamps): recompute with the generic code, patch the periodogram; whole items
            // write their partial-argmax slot (hence before the fold below), single evals fold into the running best
            SS_CUDA(cudaMemsetAsync(dmax, 0, 8 * (size_t)n_objects, stream));
            SS_CUDA(cudaMemsetAsync(dmin, 0xff, 8 * (size_t)n_objects, stream));
            ss_status_t st = launch_deferred_eval(p, defer_val, dmax, c.max_n, has_listing_options(opt), sm_count, stream);
            if (st != SS_OK) return fail(st, "deferred kernel launch failed");
            g_launches++;
        }
        fold_best_kernel<<<(unsigned)((p.n_list * 32 + 255) / 256), 256, 0, stream>>>(
            d_recs, p.list, p.n_list, (int)cpo, p.chunks_total, 0, part_val, part_idx, best_val, best_idx);
        g_launches++;
        SS_CUDA(cudaGetLastError());
        if (hands_over) {
            ss_status_t st = launch_deferred_merge(p, defer_val, dmax, dmin, best_val, best_idx, sm_count, stream);
            if (st != SS_OK) return fail(st, "deferred merge launch failed");
            g_launches += 2;
            SS_CUDA(cudaMemsetAsync(defer_count, 0, 4, stream));   // the overflow flag [1] stays
        }
    }
    // NaN rows of degenerate objects in this tile
    if (pgram && !degenerate.empty()) {
        // degenerate[] is sorted; select the sub-range inside [o0, o1)
        auto lo = std::lower_bound(degenerate.begin(), degenerate.end(), o0);
        auto hi = std::lower_bound(degenerate.begin(), degenerate.end(), o1);
        int n_rows = (int)(hi - lo);
        for (int r0 = 0; r0 < n_rows; r0 += 65535) {
            int nr = std::min(65535, n_rows - r0);
            dim3 grid((unsigned)((nk + 255) / 256), (unsigned)nr);
            nan_rows_kernel<<<grid, 256, 0, stream>>>(d_degen + (lo - degenerate.begin()) + r0, nr, row0,
                                                      nk, row_stride, pgram + (k_begin - k0));
            g_launches++;
        }
        SS_CUDA(cudaGetLastError());
    }
    return SS_OK;
}

ss_status_t Engine::finish(double* best_freq_out, int64_t* best_index_out)
{
    if (n_objects > 0 && (best_freq_out || best_index_out)) {
        finish_kernel<<<(unsigned)((n_objects + 255) / 256), 256, 0, stream>>>(n_objects, best_idx, f_min, df,
                                                                              best_freq_out, best_index_out);
        g_launches++;
        SS_CUDA(cudaGetLastError());
    }
    return SS_OK;
}

}  // namespace ss

// ================================================================================================
// C ABI
// ================================================================================================
using namespace ss;

extern "C" {

void ss_default_options(ss_options_t* opt)
{
    if (!opt) return;
    memset(opt, 0, sizeof *opt);
    opt->alpha = 9.0;
    opt->span = 0.0;
    opt->iper = 1;      // DESIGN.md R8
    opt->force_path = SS_PATH_AUTO;
}

const char* ss_last_error(void) { return g_err.c_str(); }
void ss_release_workspace(void) { ss_synchronize(); g_pool.release_all(); }
int ss_version(void) { return SS_VERSION; }
int64_t ss_last_launch_count(void) { return g_launches; }
double ss_last_kernel_ms(void) { return g_kernel_ms; }
int64_t ss_last_kernel_count(void) { return g_kernel_count; }
int ss_path_for_n(int64_t n, ss_mode_t mode) { return path_for_n(n, (int)mode); }
double ss_paper_footprint_bytes(int64_t n_t, int64_t n_f) { return paper_footprint_bytes(n_t, n_f); }
int64_t ss_paper_batches(int64_t n_t, int64_t n_f, ss_mode_t mode, double device_gib, double beta)
{
    return paper_batches(n_t, n_f, (int)mode, device_gib, beta);
}

ss_status_t ss_plan(int64_t n_points_total, int64_t max_n, int64_t n_objects, int64_t n_freq,
                    ss_mode_t mode, size_t cap_bytes, int host_tiles, int want_pgram, ss_plan_t* plan_out)
{
    if (!plan_out) return fail(SS_ERR_INVALID_ARG, "plan_out is null");
    if (n_points_total < 0 || max_n < 0 || n_objects < 0 || n_freq < 1)
        return fail(SS_ERR_INVALID_ARG, "negative size");
    PlanInput in{n_points_total, max_n, n_objects, n_freq, (int)mode, cap_bytes, host_tiles, want_pgram, 0, device_sm_count()};
    ss_status_t st = make_plan(in, plan_out);
    if (st != SS_OK) return fail(st, "cap %zu B too small", cap_bytes);
    return SS_OK;
}

size_t ss_workspace_bytes(int64_t n_points_total, int64_t max_n, int64_t n_objects, int64_t n_freq,
                          ss_mode_t mode)
{
    ss_plan_t pl{};
    PlanInput in{n_points_total, max_n, n_objects, n_freq, (int)mode, (size_t)-1, 0, 0, 0, device_sm_count()};
    if (make_plan(in, &pl) != SS_OK) return 0;
    return pl.total_bytes;
}

// One pass over the catalog with DEVICE pointers.  *overflow: the warp path's hand-over list was too short (the
// outputs are then incomplete; the caller repeats the pass on the CTA path once this pass's buffers are back in the pool).
// pending != null (asynchronous call): the engine is handed back still running instead of being waited for.
static ss_status_t periodogram_device(const double* times, const double* mags, const double* errs,
                                      const int64_t* offsets, int64_t n_objects, double f_min, double f_max,
                                      int64_t n_freq, ss_mode_t mode, double* pgram_out, double* best_freq_out,
                                      int64_t* best_index_out, const ss_options_t& o, bool* overflow,
                                      std::unique_ptr<Engine>* pending)
{
    *overflow = false;
    ss_status_t st = validate_scalars(n_objects, f_min, f_max, n_freq, (int)mode, o);
    if (st != SS_OK) return st;
    if (!offsets) return fail(SS_ERR_INVALID_ARG, "offsets is null");
    if (n_objects == 0) return SS_OK;
    cudaStream_t stream = (cudaStream_t)o.stream;
    std::vector<int64_t> off_copy;
    const int64_t* off = o.offsets_host;
    if (!off) {
        off_copy.resize((size_t)n_objects + 1);
        SS_CUDA(cudaMemcpyAsync(off_copy.data(), offsets, 8 * ((size_t)n_objects + 1), cudaMemcpyDeviceToHost, stream));
        SS_CUDA(cudaStreamSynchronize(stream));
        off = off_copy.data();
    }
    if (off[n_objects] > 0 && (!times || !mags || !errs)) return fail(SS_ERR_INVALID_ARG, "times/mags/errs is null");
    std::unique_ptr<Engine> eng(new Engine);
    st = eng->setup(times, mags, errs, off, n_objects, f_min, f_max, n_freq, (int)mode, o, false,
                    pgram_out != nullptr, 0);
    if (st != SS_OK) return st;
    // device output: the caller's array is written directly; frequency tiles only bound the
    // partial-argmax rows
    for (int ot = 0; ot < (int)eng->tiles.size(); ot++) {
        for (int64_t ft = 0; ft < eng->plan.n_freq_tiles; ft++) {
            int64_t k0 = eng->k_lo + ft * eng->plan.freq_per_tile, k1 = std::min(eng->k_lo + eng->k_n, k0 + eng->plan.freq_per_tile);
            st = eng->run_tile(ot, k0, k1, (int)ft, pgram_out, eng->k_n, 0, eng->k_lo);
            if (st != SS_OK) return st;
        }
    }
    st = eng->finish(best_freq_out, best_index_out);
    if (st != SS_OK) return st;
    if (pending) {
        *pending = std::move(eng);
        return SS_OK;
    }
    SS_CUDA(cudaStreamSynchronize(stream));
    eng->collect_profile();
    *overflow = eng->defer_overflowed();
    return SS_OK;
}

// this thread's asynchronous call in flight (ss_options_t::async_mode)
struct PendingCall {
    std::unique_ptr<Engine> eng;
    const double *times, *mags, *errs;
    const int64_t* offsets;
    std::vector<int64_t> offsets_host;
    int64_t n_objects, n_freq;
    double f_min, f_max;
    ss_mode_t mode;
    double *pgram_out, *best_freq_out;
    int64_t* best_index_out;
    ss_options_t o;
};
static thread_local std::unique_ptr<PendingCall> g_pending;

ss_status_t ss_synchronize(void)
{
    if (!g_pending) return SS_OK;
    std::unique_ptr<PendingCall> pc = std::move(g_pending);
    if (cudaStreamSynchronize((cudaStream_t)pc->o.stream) != cudaSuccess) {
        pc->eng.reset();
        return fail(SS_ERR_CUDA, "asynchronous call failed: %s", cudaGetErrorString(cudaGetLastError()));
    }
    pc->eng->collect_profile();
    const bool overflow = pc->eng->defer_overflowed();
    pc->eng.reset();                                  // workspace back to the pool
    if (!overflow) return SS_OK;
    if (pc->o.force_path == SS_PATH_BLOCK) return fail(SS_ERR_CUDA, "hand-over list overflow on the CTA path");
    ss_options_t o = pc->o;
    o.force_path = SS_PATH_BLOCK; o.async_mode = 0; o.offsets_host = pc->offsets_host.data();
    bool again = false;
    return periodogram_device(pc->times, pc->mags, pc->errs, pc->offsets, pc->n_objects, pc->f_min, pc->f_max, pc->n_freq,
                              pc->mode, pc->pgram_out, pc->best_freq_out, pc->best_index_out, o, &again, nullptr);
}

ss_status_t ss_periodogram_ex(const double* times, const double* mags, const double* errs,
                              const int64_t* offsets, int64_t n_objects, double f_min, double f_max,
                              int64_t n_freq, ss_mode_t mode, double* pgram_out, double* best_freq_out,
                              int64_t* best_index_out, const ss_options_t* opt_in)
{
    ss_status_t st = ss_synchronize();
    if (st != SS_OK) return st;
    g_launches = 0;
    ss_options_t o;
    if (opt_in) o = *opt_in; else ss_default_options(&o);
    bool overflow = false;
    if (o.async_mode) {
        if (!o.skip_validation || !o.offsets_host)
            return fail(SS_ERR_INVALID_ARG, "async_mode needs skip_validation = 1 and offsets_host");
        std::unique_ptr<PendingCall> pc(new PendingCall);
        st = periodogram_device(times, mags, errs, offsets, n_objects, f_min, f_max, n_freq, mode, pgram_out,
                                best_freq_out, best_index_out, o, &overflow, &pc->eng);
        if (st != SS_OK || !pc->eng) return st;
        pc->times = times; pc->mags = mags; pc->errs = errs; pc->offsets = offsets;
        pc->offsets_host.assign(o.offsets_host, o.offsets_host + n_objects + 1);
        pc->n_objects = n_objects; pc->n_freq = n_freq; pc->f_min = f_min; pc->f_max = f_max; pc->mode = mode;
        pc->pgram_out = pgram_out; pc->best_freq_out = best_freq_out; pc->best_index_out = best_index_out; pc->o = o;
        g_pending = std::move(pc);
        return SS_OK;
    }
    st = periodogram_device(times, mags, errs, offsets, n_objects, f_min, f_max, n_freq, mode, pgram_out,
                            best_freq_out, best_index_out, o, &overflow, nullptr);
    if (st == SS_OK && overflow) {
        // more ties than the hand-over list holds (e.g. integer time stamps at a commensurate frequency in every
        // object): serve everything with the generic kernel instead.  The first pass's buffers are already released.
        if (o.force_path == SS_PATH_BLOCK) return fail(SS_ERR_CUDA, "hand-over list overflow on the CTA path");
        o.force_path = SS_PATH_BLOCK;
        st = periodogram_device(times, mags, errs, offsets, n_objects, f_min, f_max, n_freq, mode, pgram_out,
                                best_freq_out, best_index_out, o, &overflow, nullptr);
    }
    return st;
}

ss_status_t ss_periodogram(const double* times, const double* mags, const double* errs,
                           const int64_t* offsets, int64_t n_objects, double f_min, double f_max,
                           int64_t n_freq, ss_mode_t mode, double* pgram_out, double* best_freq_out,
                           int64_t* best_index_out)
{
    return ss_periodogram_ex(times, mags, errs, offsets, n_objects, f_min, f_max, n_freq, mode, pgram_out,
                             best_freq_out, best_index_out, nullptr);
}

static ss_status_t periodogram_host(const double* times, const double* mags, const double* errs,
                                    const int64_t* offsets, int64_t n_objects, double f_min, double f_max,
                                    int64_t n_freq, ss_mode_t mode, double* pgram_out, double* best_freq_out,
                                    int64_t* best_index_out, const ss_options_t& o, bool* overflow)
{
    *overflow = false;
    ss_status_t st = validate_scalars(n_objects, f_min, f_max, n_freq, (int)mode, o);
    if (st != SS_OK) return st;
    if (!offsets) return fail(SS_ERR_INVALID_ARG, "offsets is null");
    if (n_objects == 0) return SS_OK;
    for (int64_t i = 0; i < n_objects; i++)
        if (offsets[i + 1] < offsets[i]) return fail(SS_ERR_INVALID_ARG, "offsets not non-decreasing");
    const int64_t total = offsets[n_objects];
    if (total > 0 && (!times || !mags || !errs)) return fail(SS_ERR_INVALID_ARG, "times/mags/errs is null");
    cudaStream_t stream = (cudaStream_t)o.stream;

    Engine eng;
    // raw catalog copy + best outputs live in the engine's workspace ("extra")
    const size_t raw_b = align_up(8 * (size_t)total);
    const size_t out_b = align_up(8 * (size_t)n_objects);
    // the raw copy must exist before setup() runs the prep kernel: allocate it separately first
    char* raw = nullptr;
    const size_t raw_total = 3 * raw_b + 2 * out_b + 256;
    SS_CUDA(g_pool.acquire(raw_total, &raw));
    struct Guard { char* p; size_t b; cudaStream_t s; ~Guard() { cudaStreamSynchronize(s); g_pool.release(p, b); } } guard{raw, raw_total, stream};
    double* d_t = (double*)raw; double* d_y = (double*)(raw + raw_b); double* d_e = (double*)(raw + 2 * raw_b);
    double* d_bf = (double*)(raw + 3 * raw_b); int64_t* d_bi = (int64_t*)(raw + 3 * raw_b + out_b);
    if (total > 0) {
        SS_CUDA(cudaMemcpyAsync(d_t, times, 8 * (size_t)total, cudaMemcpyHostToDevice, stream));
        SS_CUDA(cudaMemcpyAsync(d_y, mags, 8 * (size_t)total, cudaMemcpyHostToDevice, stream));
        SS_CUDA(cudaMemcpyAsync(d_e, errs, 8 * (size_t)total, cudaMemcpyHostToDevice, stream));
    }
    st = eng.setup(d_t, d_y, d_e, offsets, n_objects, f_min, f_max, n_freq, (int)mode, o, true,
                   pgram_out != nullptr, pgram_out ? 0 : 0);
    if (st != SS_OK) return st;

    // periodogram tiles: two device buffers, D2H of tile i overlaps the kernels of tile i+1
    double* tile_buf[2] = {nullptr, nullptr};
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t done[2] = {nullptr, nullptr}, copied[2] = {nullptr, nullptr};
    const size_t tile_alloc = std::max<size_t>(eng.plan.tile_bytes, 8);
    struct TileRes {
        double** b; size_t bytes; cudaEvent_t* d; cudaEvent_t* c; cudaStream_t s; cudaStream_t* cs;
        ~TileRes() {
            cudaStreamSynchronize(s);
            if (*cs) cudaStreamSynchronize(*cs);
            for (int i = 0; i < 2; i++) { g_pool.release((char*)b[i], bytes); g_pool.event_back(false, d[i]); g_pool.event_back(false, c[i]); }
        }
    } tres{tile_buf, tile_alloc, done, copied, stream, &copy_stream};
    if (pgram_out) {
        for (int i = 0; i < 2; i++) {
            char* tb_ = nullptr;
            SS_CUDA(g_pool.acquire(tile_alloc, &tb_));
            tile_buf[i] = (double*)tb_;
            SS_CUDA(g_pool.event(false, &done[i]));
            SS_CUDA(g_pool.event(false, &copied[i]));
        }
        SS_CUDA(g_pool.stream(&copy_stream));
    }
    int it = 0;
    for (int ot = 0; ot < (int)eng.tiles.size(); ot++) {
        const int64_t o0 = (int64_t)ot * eng.plan.objects_per_tile;
        const int64_t o1 = std::min(n_objects, o0 + eng.plan.objects_per_tile);
        for (int64_t ft = 0; ft < eng.plan.n_freq_tiles; ft++, it++) {
            const int64_t k0 = eng.k_lo + ft * eng.plan.freq_per_tile, k1 = std::min(eng.k_lo + eng.k_n, k0 + eng.plan.freq_per_tile);
            const int bi = it & 1;
            double* tb = pgram_out ? tile_buf[bi] : nullptr;
            if (pgram_out && it >= 2) SS_CUDA(cudaStreamWaitEvent(stream, copied[bi], 0));
            st = eng.run_tile(ot, k0, k1, (int)ft, tb, k1 - k0, o0, k0);
            if (st != SS_OK) return st;
            if (pgram_out) {
                SS_CUDA(cudaEventRecord(done[bi], stream));
                SS_CUDA(cudaStreamWaitEvent(copy_stream, done[bi], 0));
                SS_CUDA(cudaMemcpy2DAsync(pgram_out + o0 * eng.k_n + (k0 - eng.k_lo), 8 * (size_t)eng.k_n, tb, 8 * (size_t)(k1 - k0),
                                          8 * (size_t)(k1 - k0), (size_t)(o1 - o0), cudaMemcpyDeviceToHost, copy_stream));
                SS_CUDA(cudaEventRecord(copied[bi], copy_stream));
            }
        }
    }
    st = eng.finish(best_freq_out ? d_bf : nullptr, best_index_out ? d_bi : nullptr);
    if (st != SS_OK) return st;
    if (best_freq_out) SS_CUDA(cudaMemcpyAsync(best_freq_out, d_bf, 8 * (size_t)n_objects, cudaMemcpyDeviceToHost, stream));
    if (best_index_out) SS_CUDA(cudaMemcpyAsync(best_index_out, d_bi, 8 * (size_t)n_objects, cudaMemcpyDeviceToHost, stream));
    SS_CUDA(cudaStreamSynchronize(stream));
    if (copy_stream) SS_CUDA(cudaStreamSynchronize(copy_stream));
    eng.collect_profile();
    *overflow = eng.defer_overflowed();
    return SS_OK;
}

ss_status_t ss_periodogram_host(const double* times, const double* mags, const double* errs,
                                const int64_t* offsets, int64_t n_objects, double f_min, double f_max,
                                int64_t n_freq, ss_mode_t mode, double* pgram_out, double* best_freq_out,
                                int64_t* best_index_out, const ss_options_t* opt_in)
{
    ss_status_t st = ss_synchronize();
    if (st != SS_OK) return st;
    g_launches = 0;
    ss_options_t o;
    if (opt_in) o = *opt_in; else ss_default_options(&o);
    if (o.async_mode) return fail(SS_ERR_INVALID_ARG, "async_mode applies to ss_periodogram_ex only");
    bool overflow = false;
    st = periodogram_host(times, mags, errs, offsets, n_objects, f_min, f_max, n_freq, mode, pgram_out,
                                      best_freq_out, best_index_out, o, &overflow);
    if (st == SS_OK && overflow) {
        if (o.force_path == SS_PATH_BLOCK) return fail(SS_ERR_CUDA, "hand-over list overflow on the CTA path");
        o.force_path = SS_PATH_BLOCK;
        st = periodogram_host(times, mags, errs, offsets, n_objects, f_min, f_max, n_freq, mode, pgram_out,
                              best_freq_out, best_index_out, o, &overflow);
    }
    return st;
}

ss_status_t ss_debug_eval(const double* times, const double* mags, const double* errs, int64_t n,
                          double freq, ss_mode_t mode, const ss_options_t* opt_in, double* smo_out,
                          int32_t* perm_out, double* p_out)
{
    g_launches = 0;
    ss_options_t o;
    if (opt_in) o = *opt_in; else ss_default_options(&o);
    ss_status_t st = validate_scalars(1, freq, freq * 2 + 1, 1, (int)mode, o);
    if (st != SS_OK) return st;
    if (n < MIN_POINTS) return fail(SS_ERR_INVALID_ARG, "n < 5");
    if (!times || !mags || !errs) return fail(SS_ERR_INVALID_ARG, "null input");
    int64_t off[2] = {0, n};
    o.force_path = SS_PATH_STAGE;
    Engine eng;
    st = eng.setup(times, mags, errs, off, 1, freq, freq * 2 + 1, 1, (int)mode, o, false, false, 0);
    if (st != SS_OK) return st;
    EvalParams p{};
    p.tt = eng.tt; p.yc = eng.yc; p.w = eng.w; p.recs = eng.d_recs; p.alpha = o.alpha; p.mode = (int)mode;
    p.iper = o.iper; p.span = o.span;
    p.stage = eng.stage; p.stage_stride = eng.stage_stride;
    st = launch_block_debug(p, has_listing_options(o), freq, smo_out, perm_out, p_out, eng.stream);
    if (st != SS_OK) return fail(st, "debug kernel launch failed");
    g_launches++;
    SS_CUDA(cudaGetLastError());
    SS_CUDA(cudaStreamSynchronize(eng.stream));
    return SS_OK;
}

ss_status_t ss_microbench(double* fp64_flops_out, double* smem_bytes_per_s_out, void* stream_v)
{
    cudaStream_t stream = (cudaStream_t)stream_v;
    int dev = 0, sms = 0;
    SS_CUDA(cudaGetDevice(&dev));
    SS_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    double* d = nullptr;
    SS_CUDA(cudaMalloc((void**)&d, 64));
    cudaEvent_t e0, e1;
    SS_CUDA(cudaEventCreate(&e0));
    SS_CUDA(cudaEventCreate(&e1));
    const int grid = sms * 8, iters = 1 << 15;
    float ms = 0, best = 1e30f;
    for (int rep = 0; rep < 5; rep++) {
        SS_CUDA(cudaEventRecord(e0, stream));
        fp64_peak_kernel<<<grid, 256, 0, stream>>>(d, iters);
        SS_CUDA(cudaEventRecord(e1, stream));
        SS_CUDA(cudaEventSynchronize(e1));
        SS_CUDA(cudaEventElapsedTime(&ms, e0, e1));
        if (rep > 0 && ms < best) best = ms;
    }
    if (fp64_flops_out) *fp64_flops_out = 2.0 * 8.0 * (double)iters * 256.0 * grid / (best * 1e-3);
    best = 1e30f;
    for (int rep = 0; rep < 5; rep++) {
        SS_CUDA(cudaEventRecord(e0, stream));
        smem_peak_kernel<<<grid, 256, 0, stream>>>(d, iters);
        SS_CUDA(cudaEventRecord(e1, stream));
        SS_CUDA(cudaEventSynchronize(e1));
        SS_CUDA(cudaEventElapsedTime(&ms, e0, e1));
        if (rep > 0 && ms < best) best = ms;
    }
    if (smem_bytes_per_s_out) *smem_bytes_per_s_out = 8.0 * 8.0 * (double)iters * 256.0 * grid / (best * 1e-3);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(d);
    return SS_OK;
}

// ---- the entry point that allocates nothing (include/ss_periodogram.h: ss_periodogram_static) ---------------------
// The workspace of the ordinary call, carved from a built-in array instead of the pooled cudaMalloc buffer.  In HOST
// code the array's name is only a handle for the runtime, not a device address: the address every kernel is given
// comes from cudaGetSymbolAddress, asked once per device with that device current.
static __device__ __align__(256) unsigned char g_static_scratch[SS_STATIC_SCRATCH_BYTES];

constexpr int STATIC_MAX_DEVICES = 64;
constexpr unsigned int STATIC_DEFER_CAPACITY = 1u << 16;      // hand-over list of the static call: 1 MB instead of 16 MB
static std::mutex g_static_mutex;
static void* g_static_addr[STATIC_MAX_DEVICES] = {};

static ss_status_t static_scratch_address(void** out)
{
    int dev = 0;
    SS_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= STATIC_MAX_DEVICES) return fail(SS_ERR_UNSUPPORTED, "device ordinal %d (limit %d)", dev, STATIC_MAX_DEVICES);
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_addr[dev]) {
        void* ptr = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&ptr, g_static_scratch);
        if (e != cudaSuccess || !ptr)
            return fail(SS_ERR_CUDA, "cudaGetSymbolAddress of the built-in scratch failed on device %d: %s", dev, cudaGetErrorString(e));
        g_static_addr[dev] = ptr;
    }
    *out = g_static_addr[dev];
    return SS_OK;
}

ss_status_t ss_periodogram_static(const double* times, const double* mags, const double* errs,
                                  const int64_t* offsets, const int64_t* offsets_host, int64_t n_objects,
                                  double f_min, double f_max, int64_t n_freq, ss_mode_t mode,
                                  double* pgram_out, double* best_freq_out, int64_t* best_index_out, void* stream)
{
    if (!offsets_host) return fail(SS_ERR_INVALID_ARG, "ss_periodogram_static needs offsets_host");
    if (n_objects < 0 || n_freq < 1) return fail(SS_ERR_INVALID_ARG, "negative size");
    // what the call needs, from the host copy of the offsets alone: reject before anything is launched or written
    int64_t total = 0, max_n = 0;
    for (int64_t i = 0; i < n_objects; i++) {
        const int64_t n = offsets_host[i + 1] - offsets_host[i];
        if (n < 0) return fail(SS_ERR_INVALID_ARG, "offsets not non-decreasing at %lld", (long long)i);
        total += n;
        max_n = std::max(max_n, n);
    }
    ss_plan_t need{}, fit{};
    PlanInput pin{total, max_n, n_objects, n_freq, (int)mode, (size_t)-1, 0, pgram_out ? 1 : 0, 0, device_sm_count(), STATIC_DEFER_CAPACITY};
    make_plan(pin, &need);
    pin.cap_bytes = SS_STATIC_SCRATCH_BYTES;
    if (make_plan(pin, &fit) != SS_OK || fit.total_bytes > SS_STATIC_SCRATCH_BYTES)
        return fail(SS_ERR_UNSUPPORTED,
                    "ss_periodogram_static: this catalog (%lld points, longest light curve %lld) needs at least %zu B of "
                    "workspace (%zu B untiled); the built-in scratch holds %u B -- use ss_periodogram_ex",
                    (long long)total, (long long)max_n, (size_t)(need.fixed_bytes + need.stage_bytes), (size_t)need.total_bytes,
                    (unsigned)SS_STATIC_SCRATCH_BYTES);
    void* scratch = nullptr;
    ss_status_t st = static_scratch_address(&scratch);
    if (st != SS_OK) return st;
    ss_options_t o;
    ss_default_options(&o);
    o.stream = stream;
    o.workspace = scratch;
    o.workspace_bytes = SS_STATIC_SCRATCH_BYTES;
    o.workspace_cap = SS_STATIC_SCRATCH_BYTES;
    o.offsets_host = offsets_host;
    o.defer_capacity = STATIC_DEFER_CAPACITY;
    return ss_periodogram_ex(times, mags, errs, offsets, n_objects, f_min, f_max, n_freq, mode, pgram_out, best_freq_out,
                             best_index_out, &o);
}

}  // extern "C"
