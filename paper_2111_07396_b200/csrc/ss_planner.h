// ss_planner.h -- host-only logic of the batch planner and path selection (P6 in DESIGN.md).
// Pure C++ (no CUDA calls) so it can be exercised on a machine without a GPU.
#pragma once
#include <cmath>
#include <cstddef>
#include <cstdint>

#include "../../include/ss_periodogram.h"

namespace ss {

// Shared-memory budget of the BLOCK path: 14 arrays of (n+2) doubles per eval, 227 KB per CTA.
constexpr int64_t BLOCK_SMEM_MAX = 232448 - 2048;   // dynamic part; 2 KB left for static arrays
constexpr int64_t BLOCK_BYTES_PER_POINT = 14 * 8;
constexpr int64_t BLOCK_MAX_N = BLOCK_SMEM_MAX / BLOCK_BYTES_PER_POINT - 2;   // 2055

static_assert(SS_GROUP_MAX_N == BLOCK_MAX_N, "SS_GROUP_MAX_N: up to here the group path's hand-over fits the generic shared-memory kernel; beyond it uses the staging scratch");

inline int path_for_n(int64_t n, int /*mode*/)
{
    if (n <= SS_WARP_MAX_N) return SS_PATH_WARP;
    if (n <= SS_GROUP_LONG_MAX_N) return SS_PATH_GROUP;
    if (n <= SS_CLUSTER_MAX_N) return SS_PATH_CLUSTER;
    return SS_PATH_STAGE;
}

constexpr int SHARED_TIMES_M = 4;          // objects per work item of the shared-time-sampling warp kernel
constexpr int WARP_VARIANT_OPT = 2000;      // warp variant id of the listing-options kernel: WARP_VARIANT_OPT + points per lane
constexpr int GROUP_VARIANT_F32 = 1000;   // added to the group variant id: smoother scalar float (mixed precision)
constexpr int GROUP_VARIANT_OPT = 2000;   // added to the group variant id: the kernels with the listing's options compiled in
constexpr int WARP_VARIANT_F32 = 1000;    // added to the warp variant id: the same (below WARP_VARIANT_OPT)

// Cluster-path kernel variant: R CTAs of 512 threads x C points per thread, the smallest capacity R*512*C >= n
// (3,072 ... 40,960).  id = R*8 + C.
inline int cluster_variant_for_n(int n)
{
    for (int r = 2; r <= 16; r <<= 1)
        for (int c = 3; c <= 5; c++)
            if (r * 512 * c >= n) return r * 8 + c;
    return 16 * 8 + 5;
}

// Group-path kernel variant of an object: G warps x C points per thread, the smallest capacity 32*G*C >= n among
// (4,3) 384, (4,4) 512, (4,5) 640, (4,6) 768, (8,4) 1,024, (8,5) 1,280, (8,6) 1,536, (16,4) 2,048, (16,5) 2,560, and for
// SS_GROUP_MAX_N < n <= SS_GROUP_LONG_MAX_N (y, w gathered from global memory) (16,6) 3,072, (16,7) 3,584.  More
// points per thread beat more warps per eval (measured: (8,6) 2.37e10 point-evals/s at n = 1,400 where (16,3) gave
// 1.85e10; (4,6) 2.49e10 at n = 700 where (8,3) gave 2.23e10); C = 6 is what tensor memory allows at 16 warps per SM
// (20C columns per warp <= 128).  id = G*8 + C.
inline int group_variant_for_n(int n)
{
    const int gs[3] = {4, 8, 16};
    for (int gi = 0; gi < 3; gi++)
        for (int c = 3; c <= 7; c++)
            if (32 * gs[gi] * c >= n && !(gs[gi] > 4 && c == 3)) return gs[gi] * 8 + c;
    return 16 * 8 + 7;
}

// Window half-width of Friedman's smoother (O4/R21): max(2, floor(0.5*span*n + 0.5)),
// evaluated in this order in IEEE double with no contraction (volatile keeps the compiler honest).
inline int half_width(int64_t n, double span)
{
    volatile double a = 0.5 * span;
    volatile double b = a * (double)n;
    volatile double c = b + 0.5;
    int ibw = (int)std::floor(c);
    return ibw < 2 ? 2 : ibw;
}

constexpr bool WARP_IMPLEMENTED = true;
constexpr int WARPS_PER_CTA = 8;      // frequency chunks of the warp path are multiples of this

// Warp-path kernel variant of an object: (C, IBW0), C = points per lane = ceil(n/32) (at least 2), IBW0 = tweeter
// half-width (compile-time in the kernel so the halo registers are statically indexed).  id = C*8 + IBW0.
inline int warp_variant_for_n(int n)
{
    int ibw0 = half_width(n, 0.05);
    int c = (n + 31) / 32;
    if (c < 2) c = 2;
    if (c == 7 && ibw0 == 6) c = 8;      // n = 220..224: the halo of 6 needs IBW0 <= C with room; served by C = 8
    return c * 8 + ibw0;
}

// The paper's footprint model.
inline double paper_footprint_bytes(int64_t n_t, int64_t n_f) { return 15.0 * 8.0 * (double)n_t * (double)n_f; }
inline double paper_r_gib(int64_t n_t, int64_t n_f, int mode)
{
    double per = mode == SS_MODE_GENERALIZED_VALIDATION ? 96.0 : 160.0;
    return (8.0 * (double)n_f + 24.0 * (double)n_t + per * (double)n_f * (double)n_t) / (1024.0 * 1024.0 * 1024.0);
}
inline int64_t paper_batches(int64_t n_t, int64_t n_f, int mode, double device_gib, double beta)
{
    double nb = paper_r_gib(n_t, n_f, mode) / (beta * device_gib);
    int64_t b = (int64_t)std::ceil(nb);
    return b < 1 ? 1 : b;
}

constexpr unsigned int DEFER_CAPACITY = 1u << 20;   // evals the warp path may defer per tile
constexpr int DEFAULT_SM_COUNT = 148;    // B200; the planner queries take the device's own count when there is one
constexpr int64_t MIN_CHUNK = 1;          // smallest frequency chunk a work item may cover

// Work items are (object, frequency chunk).  Launches are per path class (about a tenth of a ragged catalog
// each), so aim at >= TARGET_ITEMS items per tile: the last wave of a launch is then a per-cent of it, not a
// tenth (config 3: 16,384 -> 131,072 items bought 3 % CV, 3.6 % GV; 262,144 no more).  Items keep at least 8
// frequencies each while that still leaves >= 4,096 of them (a single long light curve).
constexpr int64_t TARGET_ITEMS = 131072;
inline int64_t chunks_per_object(int64_t n_objects_in_tile, int64_t freq_per_tile)
{
    if (n_objects_in_tile < 1) n_objects_in_tile = 1;
    int64_t c = (TARGET_ITEMS + n_objects_in_tile - 1) / n_objects_in_tile;
    if (c > freq_per_tile) c = freq_per_tile;
    if (c < 1) c = 1;
    if (freq_per_tile / c < 8) {
        const int64_t c8 = freq_per_tile / 8 > 1 ? freq_per_tile / 8 : 1;
        if (c8 * n_objects_in_tile >= 4096) c = c8;
    }
    return c;
}

struct PlanInput {
    int64_t n_points_total, max_n, n_objects, n_freq;
    int mode;
    size_t cap_bytes;
    int host_tiles;    // output tiles are device buffers copied back (x2, double buffered)
    int want_pgram;
    int64_t force_freq_tile;
    int sm_count = DEFAULT_SM_COUNT;
    unsigned int defer_capacity = DEFER_CAPACITY;
};

// ---- the one workspace buffer of a call, carved: the SAME function sizes it for the planner queries (worst-case
// counts: every object kept, every object padded by one element) and for the engine (actual counts), so what
// ss_workspace_bytes() reports is an upper bound of what a call allocates or takes from the caller.
inline size_t ws_align(size_t x) { return (x + 255) / 256 * 256; }
struct WsCounts {
    int64_t padded_points = 0;   // elements of tt / yc / w (objects padded to an even length)
    int64_t n_recs = 0;          // objects with n >= 5
    int64_t n_list = 0;          // entries of the class lists
    int64_t n_degenerate = 0;    // objects with n < 5
    int64_t n_objects = 0;
    int64_t partial_slots = 0;   // (object, chunk) partial-argmax slots of one tile
    int64_t max_n = 0;
    int stage = 0;               // the global staging scratch is needed
    int sm_count = DEFAULT_SM_COUNT;
    unsigned int defer_capacity = DEFER_CAPACITY;
};
struct WsLayout {
    size_t tt, yc, w, recs, raw, list, degen, best_val, best_idx, part_val, part_idx, counters, flag, stage, defer_entries,
        defer_val, defer_count, dmax, dmin, bytes;
    int64_t stage_stride;
    int stage_ctas;
};
constexpr int WS_COUNTERS = 64;
constexpr size_t OBJREC_BYTES = 64;
inline WsLayout ws_layout(const WsCounts& c)
{
    WsLayout L{};
    size_t b = 0;
    auto carve = [&](size_t bytes) { size_t o = b; b += ws_align(bytes); return o; };
    auto atl1 = [](int64_t v) { return (size_t)(v > 1 ? v : 1); };
    L.tt = carve(8 * (size_t)c.padded_points); L.yc = carve(8 * (size_t)c.padded_points); L.w = carve(8 * (size_t)c.padded_points);
    L.recs = carve(OBJREC_BYTES * atl1(c.n_recs));
    L.raw = carve(8 * atl1(c.n_recs));
    L.list = carve(4 * atl1(c.n_list));
    L.degen = carve(8 * atl1(c.n_degenerate));
    L.best_val = carve(8 * atl1(c.n_objects)); L.best_idx = carve(8 * atl1(c.n_objects));
    L.part_val = carve(8 * atl1(c.partial_slots)); L.part_idx = carve(8 * atl1(c.partial_slots));
    L.counters = carve(4 * (size_t)WS_COUNTERS); L.flag = carve(64);
    L.stage_ctas = c.sm_count * 2;
    L.stage_stride = c.stage ? 14 * ((((int64_t)c.max_n + 2)) & ~(int64_t)1) : 0;     // BLOCK_SLOTS * block_slot_len(max_n)
    L.stage = carve(c.stage ? 8 * (size_t)L.stage_stride * (size_t)L.stage_ctas : 0);
    L.defer_entries = carve(8 * (size_t)c.defer_capacity); L.defer_val = carve(8 * (size_t)c.defer_capacity);
    L.defer_count = carve(64);
    L.dmax = carve(8 * atl1(c.n_objects)); L.dmin = carve(8 * atl1(c.n_objects));
    L.bytes = b;
    return L;
}

// New footprint model: nothing is materialised at N_t*N_f.  Fixed = catalog copy (tt, yc, w) +
// records + lists + partial argmax rows; stage = scratch of the STAGE path; tiles = periodogram
// output buffers when the caller's array lives on the host.
inline ss_status_t make_plan(const PlanInput& in, ss_plan_t* out)
{
    ss_plan_t p{};
    const int64_t nobj = in.n_objects > 0 ? in.n_objects : 0;
    // worst-case counts of the workspace (every object kept and padded by one element), partial rows added below;
    // + the raw catalog copy and the best-frequency outputs when the caller's arrays live on the host
    WsCounts wc;
    wc.padded_points = in.n_points_total + nobj; wc.n_recs = nobj; wc.n_list = nobj; wc.n_degenerate = nobj;
    wc.n_objects = nobj; wc.partial_slots = 0; wc.max_n = in.max_n; wc.stage = in.max_n > BLOCK_MAX_N;
    wc.sm_count = in.sm_count > 0 ? in.sm_count : DEFAULT_SM_COUNT; wc.defer_capacity = in.defer_capacity;
    const WsLayout wl = ws_layout(wc);
    p.stage_bytes = wc.stage ? ws_align(8 * (size_t)wl.stage_stride * (size_t)wl.stage_ctas) : 0;
    p.fixed_bytes = wl.bytes - p.stage_bytes - 2 * ws_align(8)      // the two empty partial arrays come back with partials()
                  + (in.host_tiles ? 3 * ws_align(8 * (size_t)in.n_points_total) + 2 * ws_align(8 * (size_t)(nobj > 1 ? nobj : 1)) + 256 : 0);
    // partial argmax rows of ONE tile: 16 B per (object, chunk); folded into the running best per
    // object after every tile, so they never scale with the number of tiles
    auto partials = [&](int64_t f, int64_t o) { return 2 * ws_align((size_t)8 * (size_t)(nobj > 1 ? nobj : 1) * (size_t)chunks_per_object(o, f)); };
    const size_t base = p.fixed_bytes + p.stage_bytes;
    int64_t fpt = in.n_freq, opt = nobj > 0 ? nobj : 1;
    if (in.force_freq_tile > 0 && in.force_freq_tile < fpt) fpt = in.force_freq_tile;
    if (in.host_tiles && in.want_pgram) {
        // a large output goes back in at least 4 frequency tiles even when one would fit, so that the
        // device->host copy of a tile overlaps the next tile's kernels instead of trailing the last one
        if (in.force_freq_tile <= 0 && (size_t)8 * (size_t)in.n_freq * (size_t)opt >= ((size_t)256 << 20) && in.n_freq >= 4) {
            const int64_t quarter = (in.n_freq + 3) / 4;
            if (quarter < fpt) fpt = quarter;
        }
        // exact need of an (f x o) tile: double-buffered output tile + partial rows
        auto need = [&](int64_t f, int64_t o) { return base + partials(f, o) + (size_t)2 * 8 * (size_t)f * (size_t)o; };
        // shrink the frequency tile first (the paper's N_b batches), then objects;
        // need() is non-decreasing in f and in o, so bisect
        if (need(fpt, opt) > in.cap_bytes) {
            if (need(1, opt) <= in.cap_bytes) {
                int64_t lo = 1, hi = fpt;          // need(lo) fits, need(hi) does not
                while (hi - lo > 1) {
                    int64_t mid = lo + (hi - lo) / 2;
                    if (need(mid, opt) <= in.cap_bytes) lo = mid; else hi = mid;
                }
                fpt = lo;
            } else {
                fpt = 1;
                if (need(1, 1) > in.cap_bytes) return SS_ERR_OUT_OF_MEMORY;
                int64_t lo = 1, hi = opt;
                while (hi - lo > 1) {
                    int64_t mid = lo + (hi - lo) / 2;
                    if (need(1, mid) <= in.cap_bytes) lo = mid; else hi = mid;
                }
                opt = lo;
            }
        }
        p.tile_bytes = (size_t)8 * (size_t)fpt * (size_t)opt;
    }
    p.freq_per_tile = fpt;
    p.n_freq_tiles = (in.n_freq + fpt - 1) / fpt;
    p.objects_per_tile = opt;
    p.n_object_tiles = nobj > 0 ? (nobj + opt - 1) / opt : 0;
    p.fixed_bytes += partials(fpt, opt);
    p.total_bytes = p.fixed_bytes + p.stage_bytes + (in.host_tiles && in.want_pgram ? 2 * p.tile_bytes : 0);
    if (p.total_bytes > in.cap_bytes) return SS_ERR_OUT_OF_MEMORY;
    *out = p;
    return SS_OK;
}

}  // namespace ss
