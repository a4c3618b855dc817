// spd_common.cuh -- shared declarations of the libspd kernels (sm_100a only).
// Internal to paper_1611_09704_b200/csrc; the public C ABI is include/spd.h.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>
#include <math.h>

#include "../../include/spd.h"

#if defined(__CUDA_ARCH__) && (__CUDA_ARCH__ < 1000)
#error "libspd is written for sm_100a (B200) only"
#endif

namespace spd {

// ---- Chan, Golub & LeVeque partial: m samples, T = sum, S = sum of squared deviations
struct Tri { double m, T, S; };

// eq. 2: a <- a (+) b.  Written as (n T1 - m T2)^2 / (m n (m+n)), the same quantity as the
// printed m/(n(m+n)) ((n/m) T1 - T2)^2 with one division.  A side with zero samples is skipped.
__device__ __forceinline__ void tri_merge(Tri &a, const Tri &b)
{
    if (b.m == 0.0) return;
    if (a.m == 0.0) { a = b; return; }
    double d = b.m * a.T - a.m * b.T;
    a.S = a.S + b.S + d * d / (a.m * b.m * (a.m + b.m));
    a.T += b.T;
    a.m += b.m;
}

// ---- workspace layout (bytes) -----------------------------------------------------------------------
// [0, STATS_WS)        : block partials of the stats kernels (2 * MAX_PARTIALS Tri)
// [0, table bytes)     : reciprocal sigma table of the sweep (the two calls never overlap on a stream)
constexpr int    MAX_PARTIALS = 2048;
constexpr size_t STATS_WS     = 2 * MAX_PARTIALS * sizeof(Tri);
constexpr int    NMAX_LIMIT   = 65535;

__host__ __device__ inline int round_up(int a, int b) { return (a + b - 1) / b * b; }

// ---- launchers (defined in the .cu files) ---------------------------------------------------------------
cudaError_t launch_stats(const float *x, int64_t n_dm, int64_t n_t, int64_t row_stride, int nmax_for_sigma,
                         spd_stats_t *d_stats, void *d_ws, cudaStream_t s);
cudaError_t launch_stats_rows(const float *x, int64_t n_dm, int64_t n_t, int64_t row_stride, int nmax_for_sigma,
                              spd_stats_t *d_stats_rows, void *d_ws, cudaStream_t s);
size_t stats_rows_ws_bytes(int64_t n_dm);
cudaError_t launch_stats_rows_noalloc(const float *x, int64_t n_dm, int64_t n_t, int64_t row_stride, int nmax_for_sigma,
                                      spd_stats_t *d_stats_rows, cudaStream_t s);     // partials in the library's own static array
cudaError_t launch_stats_merge(const spd_stats_t *parts, int count, spd_stats_t *out, cudaStream_t s);
cudaError_t launch_sigma_table(const spd_stats_t *d_stats, int nmax, int mode, float *d_table, cudaStream_t s,
                               int wscale = 1, int nmax_total = 0, int64_t rows = 1);
cudaError_t launch_level_stats(const spd_stats_t *st, int D, spd_stats_t *out, cudaStream_t s);
cudaError_t launch_sweep_level(const float *xl, int64_t n_dm, int64_t n_l, int64_t xl_stride, const spd_stats_t *d_stats_level,
                               const float *d_table, int w0, int wmin, int wscale, bool rc, float *snr, uint16_t *width,
                               int64_t out_stride, float *dec_out, int64_t dec_stride, cudaStream_t s);
cudaError_t launch_search_level(const float *xl, int64_t n_dm, int64_t n_l, int64_t xl_stride, const spd_stats_t *d_stats_level,
                                const float *d_table, int w0, int wmin, int wscale, bool rc, float threshold, spd_candidate_t *out,
                                unsigned long long capacity, unsigned long long *d_count, float *dec_out, int64_t dec_stride, cudaStream_t s);
bool sweep_uses_constant_table(int nmax, int mode);      // eq. 4 with nmax a multiple of 8: r_w = 1/sqrt(w) from the constant bank, no table launch
cudaError_t launch_sweep(const float *x, int64_t n_dm, int64_t n_t, int64_t row_stride, const spd_stats_t *d_stats,
                         const float *d_table, int nmax, bool rc, float *snr, uint16_t *width,
                         bool fused, float threshold, spd_candidate_t *out, unsigned long long capacity,
                         unsigned long long *d_count, cudaStream_t s, int stats_stride = 0);
cudaError_t launch_candidates(const float *snr, const uint16_t *width, int64_t n_dm, int64_t n_t, int64_t row_stride,
                              float threshold, spd_candidate_t *out, unsigned long long capacity,
                              unsigned long long *d_count, cudaStream_t s, bool zero_count = true, uint32_t t_scale = 1);
size_t sweep_table_bytes(int nmax);

// ---- warp-aggregated append of candidate records (unordered list) ------------------------------
// Every lane of the warp must call this (hit = false for lanes with nothing to add).
__device__ __forceinline__ void append_candidate(bool hit, uint32_t dm, uint32_t t, float snr, uint32_t width,
                                                 spd_candidate_t *out, unsigned long long capacity,
                                                 unsigned long long *count)
{
    unsigned mask = __ballot_sync(0xffffffffu, hit);
    if (mask == 0) return;
    int lane = threadIdx.x & 31;
    int leader = __ffs(mask) - 1;
    unsigned long long base = 0;
    if (lane == leader) base = atomicAdd(count, (unsigned long long)__popc(mask));
    base = __shfl_sync(0xffffffffu, base, leader);
    if (hit) {
        unsigned long long slot = base + __popc(mask & ((1u << lane) - 1u));
        if (slot < capacity) {
            uint4 rec = make_uint4(dm, t, __float_as_uint(snr), width);
            *reinterpret_cast<uint4 *>(out + slot) = rec;
        }
    }
}

}  // namespace spd
