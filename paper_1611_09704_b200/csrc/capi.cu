// capi.cu -- the C ABI of include/spd.h: argument checks and launches only; every step runs in the kernels.
#include "spd_common.cuh"

using namespace spd;

namespace {

constexpr int NMAX_API_LIMIT = 4096;     // shared-memory bound of the sweep / sigma_Nmax tiles

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

inline bool shape_ok(int64_t n_dm, int64_t n_t, int64_t row_stride)
{
    return n_dm >= 1 && n_t >= 1 && row_stride >= n_t && n_dm <= 0xffffffffLL && n_t <= 0xffffffffLL;
}
inline bool nmax_ok(int nmax, int64_t n_t) { return nmax >= 1 && nmax <= NMAX_API_LIMIT && (int64_t)nmax <= n_t; }

}  // namespace

extern "C" {

const char *spd_status_string(spd_status s)
{
    switch (s) {
    case SPD_OK: return "SPD_OK";
    case SPD_ERR_INVALID_ARG: return "SPD_ERR_INVALID_ARG";
    case SPD_ERR_CUDA: return "SPD_ERR_CUDA";
    case SPD_ERR_WORKSPACE: return "SPD_ERR_WORKSPACE";
    case SPD_ERR_NOALLOC_LIMIT: return "SPD_ERR_NOALLOC_LIMIT: n_dm exceeds SPD_NOALLOC_MAX_ROWS (8192 rows per spd_stats_rows_noalloc call)";
    }
    return "SPD_ERR_UNKNOWN";
}

size_t spd_workspace_bytes(int64_t n_dm, int64_t n_t, int nmax)
{
    if (n_dm < 1 || n_t < 1 || nmax < 0 || nmax > NMAX_API_LIMIT) return 0;
    size_t tab = sweep_table_bytes(nmax > 0 ? nmax : 1);
    return align_up(STATS_WS > tab ? STATS_WS : tab, 256);
}

spd_status spd_stats(const float *d_x, int64_t n_dm, int64_t n_t, int64_t row_stride, int nmax_for_sigma,
                     spd_stats_t *d_stats, void *d_ws, size_t ws_bytes, void *stream)
{
    if (!d_x || !d_stats || !d_ws || !shape_ok(n_dm, n_t, row_stride)) return SPD_ERR_INVALID_ARG;
    if (nmax_for_sigma < 0 || (nmax_for_sigma > 0 && !nmax_ok(nmax_for_sigma, n_t))) return SPD_ERR_INVALID_ARG;
    if ((reinterpret_cast<uintptr_t>(d_ws) & 15) != 0) return SPD_ERR_INVALID_ARG;
    if (ws_bytes < STATS_WS) return SPD_ERR_WORKSPACE;
    cudaError_t e = launch_stats(d_x, n_dm, n_t, row_stride, nmax_for_sigma, d_stats, d_ws, (cudaStream_t)stream);
    return e == cudaSuccess ? SPD_OK : SPD_ERR_CUDA;
}

spd_status spd_stats_merge(const spd_stats_t *d_parts, int count, spd_stats_t *d_out, void *stream)
{
    if (!d_parts || !d_out || count < 1) return SPD_ERR_INVALID_ARG;
    cudaError_t e = launch_stats_merge(d_parts, count, d_out, (cudaStream_t)stream);
    return e == cudaSuccess ? SPD_OK : SPD_ERR_CUDA;
}

spd_status spd_boxcar_snr(const float *d_x, int64_t n_dm, int64_t n_t, int64_t row_stride,
                          const spd_stats_t *d_stats, int nmax, spd_sigma_mode mode,
                          float *d_snr, uint16_t *d_width, void *d_ws, size_t ws_bytes, void *stream)
{
    if (!d_x || !d_stats || !d_snr || !d_ws || !shape_ok(n_dm, n_t, row_stride) || !nmax_ok(nmax, n_t))
        return SPD_ERR_INVALID_ARG;
    if ((int)mode < 0 || (int)mode > 2 || (reinterpret_cast<uintptr_t>(d_ws) & 15) != 0) return SPD_ERR_INVALID_ARG;
    if (ws_bytes < sweep_table_bytes(nmax)) return SPD_ERR_WORKSPACE;
    cudaStream_t s = (cudaStream_t)stream;
    float *table = reinterpret_cast<float *>(d_ws);
    const bool rc = sweep_uses_constant_table(nmax, (int)mode);
    cudaError_t e = rc ? cudaSuccess : launch_sigma_table(d_stats, nmax, (int)mode, table, s);
    if (e != cudaSuccess) return SPD_ERR_CUDA;
    e = launch_sweep(d_x, n_dm, n_t, row_stride, d_stats, table, nmax, rc, d_snr, d_width, false, 0.0f, nullptr, 0, nullptr, s);
    return e == cudaSuccess ? SPD_OK : SPD_ERR_CUDA;
}

spd_status spd_candidates(const float *d_snr, const uint16_t *d_width, int64_t n_dm, int64_t n_t, int64_t row_stride,
                          float threshold, spd_candidate_t *d_out, uint64_t capacity,
                          unsigned long long *d_count, void *stream)
{
    if (!d_snr || !d_width || !d_count || (!d_out && capacity > 0) || !shape_ok(n_dm, n_t, row_stride))
        return SPD_ERR_INVALID_ARG;
    if (threshold != threshold) return SPD_ERR_INVALID_ARG;
    cudaError_t e = launch_candidates(d_snr, d_width, n_dm, n_t, row_stride, threshold, d_out, capacity, d_count,
                                      (cudaStream_t)stream);
    return e == cudaSuccess ? SPD_OK : SPD_ERR_CUDA;
}

spd_status spd_search_fused(const float *d_x, int64_t n_dm, int64_t n_t, int64_t row_stride,
                            const spd_stats_t *d_stats, int nmax, spd_sigma_mode mode, float threshold,
                            spd_candidate_t *d_out, uint64_t capacity, unsigned long long *d_count,
                            void *d_ws, size_t ws_bytes, void *stream)
{
    if (!d_x || !d_stats || !d_count || (!d_out && capacity > 0) || !d_ws || !shape_ok(n_dm, n_t, row_stride) ||
        !nmax_ok(nmax, n_t))
        return SPD_ERR_INVALID_ARG;
    if ((int)mode < 0 || (int)mode > 2 || threshold != threshold || (reinterpret_cast<uintptr_t>(d_ws) & 15) != 0)
        return SPD_ERR_INVALID_ARG;
    if (ws_bytes < sweep_table_bytes(nmax)) return SPD_ERR_WORKSPACE;
    cudaStream_t s = (cudaStream_t)stream;
    float *table = reinterpret_cast<float *>(d_ws);
    if (cudaMemsetAsync(d_count, 0, sizeof(unsigned long long), s) != cudaSuccess) return SPD_ERR_CUDA;
    const bool rc = sweep_uses_constant_table(nmax, (int)mode);
    cudaError_t e = rc ? cudaSuccess : launch_sigma_table(d_stats, nmax, (int)mode, table, s);
    if (e != cudaSuccess) return SPD_ERR_CUDA;
    e = launch_sweep(d_x, n_dm, n_t, row_stride, d_stats, table, nmax, rc, nullptr, nullptr, true, threshold, d_out,
                     capacity, d_count, s);
    return e == cudaSuccess ? SPD_OK : SPD_ERR_CUDA;
}

// ---- one (mu, sigma) per DM row (reading A3's alternative) ---------------------------------
size_t spd_workspace_bytes_rows(int64_t n_dm, int64_t n_t, int nmax)
{
    if (n_dm < 1 || n_t < 1 || nmax < 0 || nmax > NMAX_API_LIMIT) return 0;
    const size_t tab = (size_t)n_dm * sweep_table_bytes(nmax > 0 ? nmax : 1);
    const size_t st = stats_rows_ws_bytes(n_dm);
    return align_up(st > tab ? st : tab, 256);
}

spd_status spd_stats_rows(const float *d_x, int64_t n_dm, int64_t n_t, int64_t row_stride, int nmax_for_sigma,
                          spd_stats_t *d_stats_rows, void *d_ws, size_t ws_bytes, void *stream)
{
    if (!d_x || !d_stats_rows || !d_ws || !shape_ok(n_dm, n_t, row_stride)) return SPD_ERR_INVALID_ARG;
    if (nmax_for_sigma < 0 || (nmax_for_sigma > 0 && !nmax_ok(nmax_for_sigma, n_t))) return SPD_ERR_INVALID_ARG;
    if ((reinterpret_cast<uintptr_t>(d_ws) & 15) != 0) return SPD_ERR_INVALID_ARG;
    if (ws_bytes < stats_rows_ws_bytes(n_dm)) return SPD_ERR_WORKSPACE;
    cudaError_t e = launch_stats_rows(d_x, n_dm, n_t, row_stride, nmax_for_sigma, d_stats_rows, d_ws, (cudaStream_t)stream);
    return e == cudaSuccess ? SPD_OK : SPD_ERR_CUDA;
}

// spd_stats_rows without a caller workspace: the block partials go to a static device array in stats.cu (see spd.h for
// who needs this and what it costs).  No allocation here or below; too many rows are refused before any launch.
int64_t spd_stats_rows_noalloc_max_rows(void) { return SPD_NOALLOC_MAX_ROWS; }

spd_status spd_stats_rows_noalloc(const float *d_x, int64_t n_dm, int64_t n_t, int64_t row_stride, int nmax_for_sigma,
                                  spd_stats_t *d_stats_rows, void *stream)
{
    if (!d_x || !d_stats_rows || !shape_ok(n_dm, n_t, row_stride)) return SPD_ERR_INVALID_ARG;
    if (nmax_for_sigma < 0 || (nmax_for_sigma > 0 && !nmax_ok(nmax_for_sigma, n_t))) return SPD_ERR_INVALID_ARG;
    if (n_dm > SPD_NOALLOC_MAX_ROWS) return SPD_ERR_NOALLOC_LIMIT;
    cudaError_t e = launch_stats_rows_noalloc(d_x, n_dm, n_t, row_stride, nmax_for_sigma, d_stats_rows, (cudaStream_t)stream);
    return e == cudaSuccess ? SPD_OK : SPD_ERR_CUDA;
}

spd_status spd_boxcar_snr_rows(const float *d_x, int64_t n_dm, int64_t n_t, int64_t row_stride,
                               const spd_stats_t *d_stats_rows, int nmax, spd_sigma_mode mode,
                               float *d_snr, uint16_t *d_width, void *d_ws, size_t ws_bytes, void *stream)
{
    if (!d_x || !d_stats_rows || !d_snr || !d_ws || !shape_ok(n_dm, n_t, row_stride) || !nmax_ok(nmax, n_t))
        return SPD_ERR_INVALID_ARG;
    if ((int)mode < 0 || (int)mode > 2 || (reinterpret_cast<uintptr_t>(d_ws) & 15) != 0) return SPD_ERR_INVALID_ARG;
    const bool rc = sweep_uses_constant_table(nmax, (int)mode);
    if (!rc && ws_bytes < (size_t)n_dm * sweep_table_bytes(nmax)) return SPD_ERR_WORKSPACE;
    cudaStream_t s = (cudaStream_t)stream;
    float *table = reinterpret_cast<float *>(d_ws);
    cudaError_t e = rc ? cudaSuccess : launch_sigma_table(d_stats_rows, nmax, (int)mode, table, s, 1, 0, n_dm);
    if (e != cudaSuccess) return SPD_ERR_CUDA;
    e = launch_sweep(d_x, n_dm, n_t, row_stride, d_stats_rows, table, nmax, rc, d_snr, d_width, false, 0.0f, nullptr, 0, nullptr, s, 1);
    return e == cudaSuccess ? SPD_OK : SPD_ERR_CUDA;
}

spd_status spd_search_fused_rows(const float *d_x, int64_t n_dm, int64_t n_t, int64_t row_stride,
                                 const spd_stats_t *d_stats_rows, int nmax, spd_sigma_mode mode, float threshold,
                                 spd_candidate_t *d_out, uint64_t capacity, unsigned long long *d_count,
                                 void *d_ws, size_t ws_bytes, void *stream)
{
    if (!d_x || !d_stats_rows || !d_count || (!d_out && capacity > 0) || !d_ws || !shape_ok(n_dm, n_t, row_stride) ||
        !nmax_ok(nmax, n_t))
        return SPD_ERR_INVALID_ARG;
    if ((int)mode < 0 || (int)mode > 2 || threshold != threshold || (reinterpret_cast<uintptr_t>(d_ws) & 15) != 0)
        return SPD_ERR_INVALID_ARG;
    const bool rc = sweep_uses_constant_table(nmax, (int)mode);
    if (!rc && ws_bytes < (size_t)n_dm * sweep_table_bytes(nmax)) return SPD_ERR_WORKSPACE;
    cudaStream_t s = (cudaStream_t)stream;
    float *table = reinterpret_cast<float *>(d_ws);
    if (cudaMemsetAsync(d_count, 0, sizeof(unsigned long long), s) != cudaSuccess) return SPD_ERR_CUDA;
    cudaError_t e = rc ? cudaSuccess : launch_sigma_table(d_stats_rows, nmax, (int)mode, table, s, 1, 0, n_dm);
    if (e != cudaSuccess) return SPD_ERR_CUDA;
    e = launch_sweep(d_x, n_dm, n_t, row_stride, d_stats_rows, table, nmax, rc, nullptr, nullptr, true, threshold, d_out,
                     capacity, d_count, s, 1);
    return e == cudaSuccess ? SPD_OK : SPD_ERR_CUDA;
}

// ---- decimation in time + boxcar (reading A20) ----------------------------------------------------
namespace {
inline bool dec_ok(int w0, int levels, int64_t n_t) { return (w0 == 16 || w0 == 32) && levels >= 1 && levels <= 8 && (int64_t)w0 <= n_t && (w0 << (levels - 1)) <= NMAX_API_LIMIT; }
inline int64_t dec_n(int64_t n_t, int l) { return n_t >> l; }
inline int64_t dec_off(int64_t n_t, int l) { int64_t o = 0; for (int k = 0; k < l; ++k) o += (dec_n(n_t, k) + 7) & ~(int64_t)7; return o; }
inline int64_t dec_stride(int64_t n_l) { return (n_l + 3) & ~(int64_t)3; }            // row stride of a decimated series in the workspace
}

int64_t spd_decimated_level_offset(int64_t n_t, int level)
{
    if (n_t < 1 || level < 0 || level > 8) return -1;
    return dec_off(n_t, level);                                  // level == levels gives the elements per row of the packed planes
}

size_t spd_decimated_workspace_bytes(int64_t n_dm, int64_t n_t, int w0, int levels)
{
    if (n_dm < 1 || n_t < 1 || !dec_ok(w0, levels, n_t)) return 0;
    size_t b = align_up(spd_workspace_bytes(n_dm, n_t, w0), 256) + 256;            // sigma table + one spd_stats_t for the level
    if (levels > 1) b += align_up((size_t)n_dm * (size_t)dec_stride(dec_n(n_t, 1)) * 4, 256);
    if (levels > 2) b += align_up((size_t)n_dm * (size_t)dec_stride(dec_n(n_t, 2)) * 4, 256);
    return b;
}

spd_status spd_boxcar_snr_decimated(const float *d_x, int64_t n_dm, int64_t n_t, int64_t row_stride,
                                    const spd_stats_t *d_stats, int w0, int levels, spd_sigma_mode mode,
                                    float *d_snr, uint16_t *d_width, int64_t plane_stride,
                                    void *d_ws, size_t ws_bytes, void *stream)
{
    if (!d_x || !d_stats || !d_snr || !d_width || !d_ws || !shape_ok(n_dm, n_t, row_stride) || !dec_ok(w0, levels, n_t))
        return SPD_ERR_INVALID_ARG;
    if ((int)mode < 0 || (int)mode > 2 || (reinterpret_cast<uintptr_t>(d_ws) & 255) != 0) return SPD_ERR_INVALID_ARG;
    if (plane_stride < dec_off(n_t, levels) || (plane_stride & 7) != 0) return SPD_ERR_INVALID_ARG;
    if (ws_bytes < spd_decimated_workspace_bytes(n_dm, n_t, w0, levels)) return SPD_ERR_WORKSPACE;
    cudaStream_t s = (cudaStream_t)stream;
    unsigned char *p = reinterpret_cast<unsigned char *>(d_ws);
    float *table = reinterpret_cast<float *>(p);                  p += align_up(spd_workspace_bytes(n_dm, n_t, w0), 256);
    spd_stats_t *lst = reinterpret_cast<spd_stats_t *>(p);        p += 256;
    float *buf[2] = {nullptr, nullptr};
    if (levels > 1) { buf[0] = reinterpret_cast<float *>(p); p += align_up((size_t)n_dm * (size_t)dec_stride(dec_n(n_t, 1)) * 4, 256); }
    if (levels > 2) { buf[1] = reinterpret_cast<float *>(p); }
    const int nmax_total = w0 << (levels - 1);
    const bool rc = sweep_uses_constant_table(w0, (int)mode);
    const float *src = d_x;
    int64_t src_stride = row_stride;
    for (int l = 0; l < levels; ++l) {
        const int D = 1 << l;
        const int64_t n_l = dec_n(n_t, l);
        if (n_l < 1) break;
        // the sweep of level l also writes x_{l+1} (pairwise sums of the tile it has staged anyway); the two buffers alternate
        float *nxt = nullptr;
        int64_t nxt_stride = 0;
        if (l + 1 < levels && dec_n(n_t, l + 1) >= 1) { nxt = buf[l & 1]; nxt_stride = dec_stride(dec_n(n_t, l + 1)); }
        if (launch_level_stats(d_stats, D, lst, s) != cudaSuccess) return SPD_ERR_CUDA;
        if (!rc && launch_sigma_table(d_stats, w0, (int)mode, table, s, D, nmax_total) != cudaSuccess) return SPD_ERR_CUDA;
        const int64_t off = dec_off(n_t, l);
        if (launch_sweep_level(src, n_dm, n_l, src_stride, lst, table, w0, l == 0 ? 0 : w0 / 2, D, rc, d_snr + off, d_width + off,
                               plane_stride, nxt, nxt_stride, s) != cudaSuccess) return SPD_ERR_CUDA;
        src = nxt; src_stride = nxt_stride;
    }
    return SPD_OK;
}

spd_status spd_candidates_decimated(const float *d_snr, const uint16_t *d_width, int64_t n_dm, int64_t n_t, int64_t plane_stride,
                                    int levels, float threshold, spd_candidate_t *d_out, uint64_t capacity,
                                    unsigned long long *d_count, void *stream)
{
    if (!d_snr || !d_width || !d_count || (!d_out && capacity > 0) || n_dm < 1 || n_t < 1 || levels < 1 || levels > 8)
        return SPD_ERR_INVALID_ARG;
    if (threshold != threshold || plane_stride < dec_off(n_t, levels)) return SPD_ERR_INVALID_ARG;
    for (int l = 0; l < levels; ++l) {
        const int64_t off = dec_off(n_t, l), n_l = dec_n(n_t, l);
        if (n_l < 1) break;
        if (launch_candidates(d_snr + off, d_width + off, n_dm, n_l, plane_stride, threshold, d_out, capacity, d_count,
                              (cudaStream_t)stream, l == 0, 1u << l) != cudaSuccess) return SPD_ERR_CUDA;
    }
    return SPD_OK;
}

spd_status spd_search_fused_decimated(const float *d_x, int64_t n_dm, int64_t n_t, int64_t row_stride,
                                      const spd_stats_t *d_stats, int w0, int levels, spd_sigma_mode mode, float threshold,
                                      spd_candidate_t *d_out, uint64_t capacity, unsigned long long *d_count,
                                      void *d_ws, size_t ws_bytes, void *stream)
{
    if (!d_x || !d_stats || !d_count || (!d_out && capacity > 0) || !d_ws || !shape_ok(n_dm, n_t, row_stride) || !dec_ok(w0, levels, n_t))
        return SPD_ERR_INVALID_ARG;
    if ((int)mode < 0 || (int)mode > 2 || threshold != threshold || (reinterpret_cast<uintptr_t>(d_ws) & 255) != 0) return SPD_ERR_INVALID_ARG;
    if (ws_bytes < spd_decimated_workspace_bytes(n_dm, n_t, w0, levels)) return SPD_ERR_WORKSPACE;
    cudaStream_t s = (cudaStream_t)stream;
    unsigned char *p = reinterpret_cast<unsigned char *>(d_ws);
    float *table = reinterpret_cast<float *>(p);                  p += align_up(spd_workspace_bytes(n_dm, n_t, w0), 256);
    spd_stats_t *lst = reinterpret_cast<spd_stats_t *>(p);        p += 256;
    float *buf[2] = {nullptr, nullptr};
    if (levels > 1) { buf[0] = reinterpret_cast<float *>(p); p += align_up((size_t)n_dm * (size_t)dec_stride(dec_n(n_t, 1)) * 4, 256); }
    if (levels > 2) { buf[1] = reinterpret_cast<float *>(p); }
    const int nmax_total = w0 << (levels - 1);
    const bool rc = sweep_uses_constant_table(w0, (int)mode);
    if (cudaMemsetAsync(d_count, 0, sizeof(unsigned long long), s) != cudaSuccess) return SPD_ERR_CUDA;
    const float *src = d_x;
    int64_t src_stride = row_stride;
    for (int l = 0; l < levels; ++l) {
        const int D = 1 << l;
        const int64_t n_l = dec_n(n_t, l);
        if (n_l < 1) break;
        float *nxt = nullptr;                                     // the search of level l also writes x_{l+1}; the two buffers alternate
        int64_t nxt_stride = 0;
        if (l + 1 < levels && dec_n(n_t, l + 1) >= 1) { nxt = buf[l & 1]; nxt_stride = dec_stride(dec_n(n_t, l + 1)); }
        if (launch_level_stats(d_stats, D, lst, s) != cudaSuccess) return SPD_ERR_CUDA;
        if (!rc && launch_sigma_table(d_stats, w0, (int)mode, table, s, D, nmax_total) != cudaSuccess) return SPD_ERR_CUDA;
        if (launch_search_level(src, n_dm, n_l, src_stride, lst, table, w0, l == 0 ? 0 : w0 / 2, D, rc, threshold, d_out, capacity,
                                d_count, nxt, nxt_stride, s) != cudaSuccess) return SPD_ERR_CUDA;
        src = nxt; src_stride = nxt_stride;
    }
    return SPD_OK;
}

// arena layout of spd_search_host: x | candidates | stats | count | workspace
size_t spd_search_host_arena_bytes(int64_t n_dm, int64_t n_t, int nmax, uint64_t capacity)
{
    if (n_dm < 1 || n_t < 1 || nmax < 1 || nmax > NMAX_API_LIMIT) return 0;
    const size_t n = (size_t)n_dm * (size_t)n_t;
    return align_up(n * 4, 256) + align_up((size_t)capacity * sizeof(spd_candidate_t), 256) + 256 + 256 +
           spd_workspace_bytes(n_dm, n_t, nmax);
}

spd_status spd_search_host(const float *h_x, int64_t n_dm, int64_t n_t, int nmax, spd_sigma_mode mode,
                           float threshold, spd_candidate_t *h_out, uint64_t capacity,
                           unsigned long long *h_count, spd_stats_t *h_stats,
                           void *d_arena, size_t arena_bytes, void *stream)
{
    if (!h_x || !h_count || (!h_out && capacity > 0) || !d_arena || !shape_ok(n_dm, n_t, n_t) || !nmax_ok(nmax, n_t))
        return SPD_ERR_INVALID_ARG;
    if ((reinterpret_cast<uintptr_t>(d_arena) & 255) != 0) return SPD_ERR_INVALID_ARG;
    if (arena_bytes < spd_search_host_arena_bytes(n_dm, n_t, nmax, capacity)) return SPD_ERR_WORKSPACE;
    cudaStream_t s = (cudaStream_t)stream;
    const size_t n = (size_t)n_dm * (size_t)n_t;
    unsigned char *p = reinterpret_cast<unsigned char *>(d_arena);
    float *d_x = reinterpret_cast<float *>(p);                 p += align_up(n * 4, 256);
    spd_candidate_t *d_out = reinterpret_cast<spd_candidate_t *>(p); p += align_up((size_t)capacity * sizeof(spd_candidate_t), 256);
    spd_stats_t *d_stats = reinterpret_cast<spd_stats_t *>(p); p += 256;
    unsigned long long *d_count = reinterpret_cast<unsigned long long *>(p); p += 256;
    void *d_ws = p;
    const size_t ws_bytes = spd_workspace_bytes(n_dm, n_t, nmax);

    if (cudaMemcpyAsync(d_x, h_x, n * 4, cudaMemcpyHostToDevice, s) != cudaSuccess) return SPD_ERR_CUDA;
    spd_status st = spd_stats(d_x, n_dm, n_t, n_t, mode == SPD_SIGMA_SQRT ? 0 : nmax, d_stats, d_ws, ws_bytes, stream);
    if (st != SPD_OK) return st;
    st = spd_search_fused(d_x, n_dm, n_t, n_t, d_stats, nmax, mode, threshold, d_out, capacity, d_count, d_ws, ws_bytes, stream);
    if (st != SPD_OK) return st;
    if (h_stats && cudaMemcpyAsync(h_stats, d_stats, sizeof(spd_stats_t), cudaMemcpyDeviceToHost, s) != cudaSuccess) return SPD_ERR_CUDA;
    if (cudaMemcpyAsync(h_count, d_count, sizeof(unsigned long long), cudaMemcpyDeviceToHost, s) != cudaSuccess) return SPD_ERR_CUDA;
    // the first records travel with the count (64 KiB at most), so a short list costs one synchronisation, not two
    const unsigned long long spec = capacity < 4096 ? capacity : 4096;
    if (spec > 0 && cudaMemcpyAsync(h_out, d_out, (size_t)spec * sizeof(spd_candidate_t), cudaMemcpyDeviceToHost, s) != cudaSuccess) return SPD_ERR_CUDA;
    if (cudaStreamSynchronize(s) != cudaSuccess) return SPD_ERR_CUDA;
    const unsigned long long got = *h_count < capacity ? *h_count : capacity;     // (UINT64_MAX, the sigma_N sentinel, has written no record)
    if (*h_count != ~0ULL && got > spec) {
        if (cudaMemcpyAsync(h_out + spec, d_out + spec, (size_t)(got - spec) * sizeof(spd_candidate_t), cudaMemcpyDeviceToHost, s) != cudaSuccess) return SPD_ERR_CUDA;
        if (cudaStreamSynchronize(s) != cudaSuccess) return SPD_ERR_CUDA;
    }
    return SPD_OK;
}

// arena layout of spd_search_host_decimated: x | candidates | stats | count | workspace of the decimated search (which
// covers the statistics' workspace: it starts with spd_workspace_bytes(.., w0) >= STATS_WS bytes)
size_t spd_search_host_decimated_arena_bytes(int64_t n_dm, int64_t n_t, int w0, int levels, uint64_t capacity)
{
    const size_t ws = spd_decimated_workspace_bytes(n_dm, n_t, w0, levels);
    if (ws == 0) return 0;
    const size_t n = (size_t)n_dm * (size_t)n_t;
    return align_up(n * 4, 256) + align_up((size_t)capacity * sizeof(spd_candidate_t), 256) + 256 + 256 + ws;
}

spd_status spd_search_host_decimated(const float *h_x, int64_t n_dm, int64_t n_t, int w0, int levels, spd_sigma_mode mode,
                                     float threshold, spd_candidate_t *h_out, uint64_t capacity,
                                     unsigned long long *h_count, spd_stats_t *h_stats,
                                     void *d_arena, size_t arena_bytes, void *stream)
{
    if (!h_x || !h_count || (!h_out && capacity > 0) || !d_arena || !shape_ok(n_dm, n_t, n_t) || !dec_ok(w0, levels, n_t))
        return SPD_ERR_INVALID_ARG;
    if ((int)mode < 0 || (int)mode > 2 || (reinterpret_cast<uintptr_t>(d_arena) & 255) != 0) return SPD_ERR_INVALID_ARG;
    if (arena_bytes < spd_search_host_decimated_arena_bytes(n_dm, n_t, w0, levels, capacity)) return SPD_ERR_WORKSPACE;
    cudaStream_t s = (cudaStream_t)stream;
    const size_t n = (size_t)n_dm * (size_t)n_t;
    unsigned char *p = reinterpret_cast<unsigned char *>(d_arena);
    float *d_x = reinterpret_cast<float *>(p);                 p += align_up(n * 4, 256);
    spd_candidate_t *d_out = reinterpret_cast<spd_candidate_t *>(p); p += align_up((size_t)capacity * sizeof(spd_candidate_t), 256);
    spd_stats_t *d_stats = reinterpret_cast<spd_stats_t *>(p); p += 256;
    unsigned long long *d_count = reinterpret_cast<unsigned long long *>(p); p += 256;
    void *d_ws = p;
    const size_t ws_bytes = spd_decimated_workspace_bytes(n_dm, n_t, w0, levels);
    const int nmax_total = w0 << (levels - 1);

    if (cudaMemcpyAsync(d_x, h_x, n * 4, cudaMemcpyHostToDevice, s) != cudaSuccess) return SPD_ERR_CUDA;
    spd_status st = spd_stats(d_x, n_dm, n_t, n_t, mode == SPD_SIGMA_SQRT ? 0 : nmax_total, d_stats, d_ws, ws_bytes, stream);
    if (st != SPD_OK) return st;
    st = spd_search_fused_decimated(d_x, n_dm, n_t, n_t, d_stats, w0, levels, mode, threshold, d_out, capacity, d_count, d_ws, ws_bytes, stream);
    if (st != SPD_OK) return st;
    if (h_stats && cudaMemcpyAsync(h_stats, d_stats, sizeof(spd_stats_t), cudaMemcpyDeviceToHost, s) != cudaSuccess) return SPD_ERR_CUDA;
    if (cudaMemcpyAsync(h_count, d_count, sizeof(unsigned long long), cudaMemcpyDeviceToHost, s) != cudaSuccess) return SPD_ERR_CUDA;
    const unsigned long long spec = capacity < 4096 ? capacity : 4096;           // as spd_search_host: one synchronisation for a short list
    if (spec > 0 && cudaMemcpyAsync(h_out, d_out, (size_t)spec * sizeof(spd_candidate_t), cudaMemcpyDeviceToHost, s) != cudaSuccess) return SPD_ERR_CUDA;
    if (cudaStreamSynchronize(s) != cudaSuccess) return SPD_ERR_CUDA;
    const unsigned long long got = *h_count < capacity ? *h_count : capacity;
    if (*h_count != ~0ULL && got > spec) {
        if (cudaMemcpyAsync(h_out + spec, d_out + spec, (size_t)(got - spec) * sizeof(spd_candidate_t), cudaMemcpyDeviceToHost, s) != cudaSuccess) return SPD_ERR_CUDA;
        if (cudaStreamSynchronize(s) != cudaSuccess) return SPD_ERR_CUDA;
    }
    return SPD_OK;
}

}  // extern "C"
