// ss_peaks.cu -- top-k peaks of periodogram rows (include/ss_periodogram.h: ss_periodogram_peaks*).
// One CTA per row: every thread scans a contiguous segment for local maxima and keeps its own n_peaks best in
// registers, then the CTA selects the n_peaks best of the 256 sorted lists by n_peaks rounds of a block-wide argmax.
#include <algorithm>
#include <cmath>
#include <vector>

#include "../../include/ss_periodogram.h"
#include "ss_common.cuh"

namespace ss {

constexpr int PEAK_T = 256;

// (power, index) order of the result: higher power first, equal powers by lower index
__device__ __forceinline__ bool peak_before(double va, int64_t ia, double vb, int64_t ib)
{
    return va > vb || (va == vb && ia < ib);
}

template <int KP>
__global__ void __launch_bounds__(PEAK_T) peaks_kernel(const double* __restrict__ pgram, int64_t n_freq, int64_t row_stride,
                                                       double f_min, double df, int n_peaks, int64_t* peak_index_out,
                                                       double* peak_power_out, double* peak_freq_out)
{
    __shared__ double s_val[PEAK_T / 32];
    __shared__ int64_t s_idx[PEAK_T / 32];
    __shared__ int s_own[PEAK_T / 32];
    __shared__ int s_winner;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const double* row = pgram + (int64_t)blockIdx.x * row_stride;
    const int64_t seg = (n_freq + PEAK_T - 1) / PEAK_T;
    const int64_t a = (int64_t)tid * seg, b = min(a + seg, n_freq);

    // this thread's best KP peaks, sorted (registers; -inf / INT64_MAX = empty)
    double val[KP];
    int64_t idx[KP];
#pragma unroll
    for (int i = 0; i < KP; i++) { val[i] = -INFINITY; idx[i] = INT64_MAX; }
    if (a < b) {
        double prev = a > 0 ? row[a - 1] : -INFINITY;      // a neighbour outside the grid does not disqualify
        double cur = row[a];
        for (int64_t k = a; k < b; k++) {
            const double next = k + 1 < n_freq ? row[k + 1] : -INFINITY;
            if (cur > prev && cur >= next) {
                // insert (cur, k): the list stays sorted; k rises, so an equal power goes behind
                double v = cur;
                int64_t j = k;
#pragma unroll
                for (int i = 0; i < KP; i++) {
                    if (peak_before(v, j, val[i], idx[i])) {
                        const double tv = val[i]; val[i] = v; v = tv;
                        const int64_t tj = idx[i]; idx[i] = j; j = tj;
                    }
                }
            }
            prev = cur; cur = next;
        }
    }
    // n_peaks rounds: the best head of the 256 lists wins and its owner moves on
    int64_t* oi = peak_index_out + (int64_t)blockIdx.x * n_peaks;
    double* ov = peak_power_out ? peak_power_out + (int64_t)blockIdx.x * n_peaks : nullptr;
    double* of = peak_freq_out ? peak_freq_out + (int64_t)blockIdx.x * n_peaks : nullptr;
    for (int r = 0; r < n_peaks; r++) {
        double hv = val[0];
        int64_t hi = idx[0];
        int own = tid;
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) {
            const double ov2 = __shfl_xor_sync(0xffffffffu, hv, d);
            const int64_t oi2 = __shfl_xor_sync(0xffffffffu, hi, d);
            const int oo = __shfl_xor_sync(0xffffffffu, own, d);
            if (peak_before(ov2, oi2, hv, hi)) { hv = ov2; hi = oi2; own = oo; }
        }
        if (lane == 0) { s_val[warp] = hv; s_idx[warp] = hi; s_own[warp] = own; }
        __syncthreads();
        if (tid == 0) {
            for (int q = 1; q < PEAK_T / 32; q++)
                if (peak_before(s_val[q], s_idx[q], hv, hi)) { hv = s_val[q]; hi = s_idx[q]; own = s_own[q]; }
            const bool some = hi != INT64_MAX;
            oi[r] = some ? hi : -1;
            if (ov) ov[r] = some ? hv : nan("");
            if (of) of[r] = some ? freq_of(f_min, df, hi) : nan("");
            s_winner = some ? own : -1;
        }
        __syncthreads();
        if (tid == s_winner) {
#pragma unroll
            for (int i = 0; i + 1 < KP; i++) { val[i] = val[i + 1]; idx[i] = idx[i + 1]; }
            val[KP - 1] = -INFINITY; idx[KP - 1] = INT64_MAX;
        }
    }
}

static ss_status_t launch_peaks(const double* pgram, int64_t n_objects, int64_t n_freq, int64_t row_stride, double f_min,
                                double f_max, int n_peaks, int64_t* pi, double* pv, double* pf, cudaStream_t stream)
{
    const double df = (f_max - f_min) / (double)n_freq;
    for (int64_t o0 = 0; o0 < n_objects; o0 += 1 << 30) {
        const unsigned g = (unsigned)std::min<int64_t>(n_objects - o0, 1 << 30);
        const double* pg = pgram + o0 * row_stride;
        int64_t* qi = pi + o0 * n_peaks;
        double* qv = pv ? pv + o0 * n_peaks : nullptr;
        double* qf = pf ? pf + o0 * n_peaks : nullptr;
        if (n_peaks <= 4) peaks_kernel<4><<<g, PEAK_T, 0, stream>>>(pg, n_freq, row_stride, f_min, df, n_peaks, qi, qv, qf);
        else if (n_peaks <= 8) peaks_kernel<8><<<g, PEAK_T, 0, stream>>>(pg, n_freq, row_stride, f_min, df, n_peaks, qi, qv, qf);
        else if (n_peaks <= 16) peaks_kernel<16><<<g, PEAK_T, 0, stream>>>(pg, n_freq, row_stride, f_min, df, n_peaks, qi, qv, qf);
        else peaks_kernel<32><<<g, PEAK_T, 0, stream>>>(pg, n_freq, row_stride, f_min, df, n_peaks, qi, qv, qf);
    }
    return cudaGetLastError() == cudaSuccess ? SS_OK : SS_ERR_CUDA;
}

static bool peaks_args_ok(const double* pgram, int64_t n_objects, int64_t n_freq, int64_t row_stride, double f_min,
                          double f_max, int n_peaks, const int64_t* pi)
{
    return n_objects >= 0 && n_freq >= 1 && row_stride >= n_freq && n_peaks >= 1 && n_peaks <= SS_MAX_PEAKS && pi &&
           (pgram || n_objects == 0) && std::isfinite(f_min) && std::isfinite(f_max) && f_max > f_min;
}

}  // namespace ss

using namespace ss;

extern "C" {

ss_status_t ss_periodogram_peaks(const double* pgram, int64_t n_objects, int64_t n_freq, int64_t row_stride,
                                 double f_min, double f_max, int n_peaks, int64_t* peak_index_out,
                                 double* peak_power_out, double* peak_freq_out, void* stream_v)
{
    if (!peaks_args_ok(pgram, n_objects, n_freq, row_stride, f_min, f_max, n_peaks, peak_index_out)) return SS_ERR_INVALID_ARG;
    if (n_objects == 0) return SS_OK;
    cudaStream_t stream = (cudaStream_t)stream_v;
    ss_status_t st = launch_peaks(pgram, n_objects, n_freq, row_stride, f_min, f_max, n_peaks, peak_index_out,
                                  peak_power_out, peak_freq_out, stream);
    if (st != SS_OK) return st;
    return cudaStreamSynchronize(stream) == cudaSuccess ? SS_OK : SS_ERR_CUDA;
}

ss_status_t ss_periodogram_peaks_host(const double* pgram, int64_t n_objects, int64_t n_freq, int64_t row_stride,
                                      double f_min, double f_max, int n_peaks, int64_t* peak_index_out,
                                      double* peak_power_out, double* peak_freq_out)
{
    if (!peaks_args_ok(pgram, n_objects, n_freq, row_stride, f_min, f_max, n_peaks, peak_index_out)) return SS_ERR_INVALID_ARG;
    if (n_objects == 0) return SS_OK;
    // slabs of rows of at most 256 MB
    const int64_t rows = std::max<int64_t>(1, std::min<int64_t>(n_objects, ((int64_t)256 << 20) / (8 * n_freq)));
    double *d_pg = nullptr, *d_pv = nullptr, *d_pf = nullptr;
    int64_t* d_pi = nullptr;
    ss_status_t st = SS_OK;
    if (cudaMalloc((void**)&d_pg, 8 * (size_t)rows * (size_t)n_freq) != cudaSuccess ||
        cudaMalloc((void**)&d_pi, 8 * (size_t)rows * n_peaks) != cudaSuccess ||
        cudaMalloc((void**)&d_pv, 8 * (size_t)rows * n_peaks) != cudaSuccess ||
        cudaMalloc((void**)&d_pf, 8 * (size_t)rows * n_peaks) != cudaSuccess)
        st = SS_ERR_OUT_OF_MEMORY;
    for (int64_t o0 = 0; st == SS_OK && o0 < n_objects; o0 += rows) {
        const int64_t nr = std::min(rows, n_objects - o0);
        cudaError_t e = cudaMemcpy2D(d_pg, 8 * (size_t)n_freq, pgram + o0 * row_stride, 8 * (size_t)row_stride,
                                     8 * (size_t)n_freq, (size_t)nr, cudaMemcpyHostToDevice);
        if (e != cudaSuccess) { st = SS_ERR_CUDA; break; }
        st = launch_peaks(d_pg, nr, n_freq, n_freq, f_min, f_max, n_peaks, d_pi, d_pv, d_pf, nullptr);
        if (st != SS_OK) break;
        const size_t ob = 8 * (size_t)nr * n_peaks;
        if (cudaMemcpy(peak_index_out + o0 * n_peaks, d_pi, ob, cudaMemcpyDeviceToHost) != cudaSuccess) st = SS_ERR_CUDA;
        if (peak_power_out && cudaMemcpy(peak_power_out + o0 * n_peaks, d_pv, ob, cudaMemcpyDeviceToHost) != cudaSuccess) st = SS_ERR_CUDA;
        if (peak_freq_out && cudaMemcpy(peak_freq_out + o0 * n_peaks, d_pf, ob, cudaMemcpyDeviceToHost) != cudaSuccess) st = SS_ERR_CUDA;
    }
    cudaFree(d_pg); cudaFree(d_pi); cudaFree(d_pv); cudaFree(d_pf);
    return st;
}

}  // extern "C"
