/*
 * spd.h -- C ABI of libspd: single-pulse detection on de-dispersed data, native to NVIDIA B200 (sm_100a).
 *
 * Method: K. Adamek & W. Armour, "A Real-time Single Pulse Detection Algorithm for GPUs",
 * arXiv 1611.09704.  Citations are lines of /root/reference/PAPER.md ("PAPER.md:NN") plus section.
 *
 * Data: x is float32 [n_dm][n_t], row-major, time fastest ("de-dispersed time series data",
 * PAPER.md:15; one row per DM trial).  row_stride is in ELEMENTS, >= n_t, and is shared
 * by x and by the snr / width planes.
 *
 * Ownership: the caller owns every buffer, including the workspace; the library allocates nothing
 * and keeps no state.  Unless a parameter is named h_*, every pointer is a DEVICE pointer.
 * Asynchrony: every spd_* call that takes a stream only enqueues work on it and returns; it never
 * synchronises (spd_search_host is the one exception, see there).
 * Errors: return code only.  Argument checks -> SPD_ERR_INVALID_ARG; short workspace ->
 * SPD_ERR_WORKSPACE; launch / runtime failure -> SPD_ERR_CUDA.  There is no CPU fallback.
 * Undefined input: non-finite samples; sigma = 0.
 */
#ifndef SPD_H
#define SPD_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum { SPD_OK = 0, SPD_ERR_INVALID_ARG = 1, SPD_ERR_CUDA = 2, SPD_ERR_WORKSPACE = 3,
               SPD_ERR_NOALLOC_LIMIT = 4   /* spd_stats_rows_noalloc only: more rows than its built-in scratch holds */
} spd_status;

/* sigma after an N-sample boxcar (section 2.2) */
typedef enum {
    SPD_SIGMA_SQRT = 0,            /* eq. 4: sigma_N = sqrt(N) sigma */
    SPD_SIGMA_LINEAR = 1,          /* eq. 5 exactly as printed: sqrt(N) sigma + (N-1) sigma_Nmax/(Nmax-1) */
    SPD_SIGMA_LINEAR_ANCHORED = 2  /* not in the paper: sqrt(N) sigma + (N-1)(sigma_Nmax - sqrt(Nmax) sigma)/(Nmax-1) */
} spd_sigma_mode;

/* Result of spd_stats, in DEVICE memory (80 bytes).  (n, T, S) and (n_b, T_b, S_b) are the raw Chan
 * triples so that several results can be merged with eq. 2 (spd_stats_merge).
 * sigma_nmax = NaN, nmax_of_sigma = 0 when the sigma_Nmax pass was skipped. */
typedef struct {
    double   mean;           /* mu = T/n */
    double   sigma;          /* sigma = sqrt(S/n), population form */
    double   sigma_nmax;     /* std of the Nmax-sample boxcar SUMS over all full windows */
    double   T, S;           /* sum, sum of squared deviations of the samples */
    double   T_b, S_b;       /* the same for the boxcar sums */
    uint64_t n;              /* number of samples */
    uint64_t n_b;            /* number of boxcar sums: n_dm * (n_t - nmax + 1) */
    int32_t  nmax_of_sigma;  /* the Nmax sigma_nmax was measured for */
    int32_t  _pad;
} spd_stats_t;

/* One detection ("dispersion measure (DM) and the time at which an event was detected,
 * its SNR and the width of the boxcar responsible").  dm = row index, t = index of the FIRST sample of
 * the best boxcar; physical DM and time are a caller-side affine map.  16 bytes, one 128-bit store. */
typedef struct { uint32_t dm, t; float snr; uint32_t width; } spd_candidate_t;

const char *spd_status_string(spd_status s);

/* Bytes of device workspace spd_stats / spd_boxcar_snr need for this shape (the larger of the two).
 * Returns 0 for invalid arguments. */
size_t spd_workspace_bytes(int64_t n_dm, int64_t n_t, int nmax);

/* Step 1 -- mean and standard deviation (section 2.1).
 * Kernel 1 cuts the array into equal blocks; each thread runs the streaming update eq. 1 over a fixed
 * run and partial (n,T,S) are merged with eq. 2 inside the block; kernel 2 merges the block partials
 * with eq. 2 in a fixed order (bit-reproducible) and writes *d_stats.
 * nmax_for_sigma > 0 also measures the "true" sigma_Nmax that eq. 5 needs; 0 skips it.
 * Requires 1 <= n_dm, 1 <= n_t, row_stride >= n_t, 0 <= nmax_for_sigma <= min(n_t, 4096).
 * d_ws: workspace of >= spd_workspace_bytes() bytes, 16-byte aligned; contents need not persist. */
spd_status spd_stats(const float *d_x, int64_t n_dm, int64_t n_t, int64_t row_stride,
                     int nmax_for_sigma, spd_stats_t *d_stats,
                     void *d_ws, size_t ws_bytes, void *stream);

/* eq. 2 over `count` results of spd_stats on disjoint row blocks, folded in index
 * order into *d_out (mean / sigma / sigma_nmax recomputed).  This is the one exchange step of a
 * DM-row-sharded run: all-gather the 80-byte structs, then merge locally in rank order.
 * d_parts and d_out are device pointers; d_out may alias d_parts[0]. */
spd_status spd_stats_merge(const spd_stats_t *d_parts, int count, spd_stats_t *d_out, void *stream);

/* Steps 2-4a -- boxcars of every width 1..nmax, SNR, max and arg-max over width, in one kernel
 * (section 2.3, Algorithm 1 as read in DESIGN.md):
 *   B_N(t) = sum_{k<N} x[d][t+k],  SNR_N(t) = (B_N(t) - N mu) / sigma_N,  widths with t+N <= n_t only;
 *   d_snr[d][t] = max_N SNR_N(t),  d_width[d][t] = the smallest N attaining it.
 * mu, sigma (and sigma_nmax for the LINEAR modes) are read from *d_stats on the device; a LINEAR mode
 * fed stats whose nmax_of_sigma != nmax yields an all-NaN SNR plane (it cannot be caught without a sync).
 * Widths whose fp32 SNRs differ by less than about 4e-6 relative (rounding of the running sums) count as tied and
 * either may be reported; an exact tie of a non-negative maximum reports the smallest width (of a negative maximum:
 * one of the tied widths).  d_snr is always the maximum itself.
 * Requires 1 <= nmax <= min(n_t, 4096) (shared-memory bound of the tile).  d_width may be NULL (plane not written). */
spd_status spd_boxcar_snr(const float *d_x, int64_t n_dm, int64_t n_t, int64_t row_stride,
                          const spd_stats_t *d_stats, int nmax, spd_sigma_mode mode,
                          float *d_snr, uint16_t *d_width,
                          void *d_ws, size_t ws_bytes, void *stream);

/* Step 4b -- candidate selection (section 2.4): every (d,t) with d_snr[d][t] >= threshold
 * becomes one record; the planes are not modified; the list is unordered.
 * *d_count is zeroed by the call and counts ALL hits; only the first `capacity` reservations are written,
 * so the caller detects overflow as *d_count > capacity after its own synchronisation. */
spd_status spd_candidates(const float *d_snr, const uint16_t *d_width, int64_t n_dm, int64_t n_t, int64_t row_stride,
                          float threshold, spd_candidate_t *d_out, uint64_t capacity,
                          unsigned long long *d_count, void *stream);

/* Steps 2-4 fused: the sweep of spd_boxcar_snr with the threshold of spd_candidates applied in the
 * same kernel; the SNR / width planes are never written (the list is the only downstream product,
 * PAPER.md:93).  Same (dm, t, snr) as spd_boxcar_snr + spd_candidates, bit for bit; the width of a hit is found by
 * replaying its running sums, so it is the exact smallest arg-max of the fp32 values and can differ from the plane
 * path's width only inside the near-ties described there.  *d_count / capacity follow spd_candidates.
 * A LINEAR mode fed stats whose nmax_of_sigma != nmax has no sigma_N: the call then sets *d_count = UINT64_MAX
 * (no record is written), since "no detections" would be indistinguishable from the misuse. */
spd_status spd_search_fused(const float *d_x, int64_t n_dm, int64_t n_t, int64_t row_stride,
                            const spd_stats_t *d_stats, int nmax, spd_sigma_mode mode, float threshold,
                            spd_candidate_t *d_out, uint64_t capacity, unsigned long long *d_count,
                            void *d_ws, size_t ws_bytes, void *stream);

/* Per-DM-row statistics ("for the dataset": reading A3 takes one estimate per call over everything passed
 * in; one estimate per DM trial is the alternative heterogeneous data wants).
 * spd_stats_rows writes d_stats_rows[n_dm], one spd_stats_t per row (same kernels and precision as spd_stats, one row per
 * grid slice); spd_boxcar_snr_rows / spd_search_fused_rows are spd_boxcar_snr / spd_search_fused with mu, sigma (and
 * sigma_nmax) of row d taken from d_stats_rows[d].  d_ws: >= spd_workspace_bytes_rows() bytes, 16-byte aligned (block
 * partials of the statistics; one r_w table per row in the eq. 5 modes).  A row with sigma = 0 is undefined input. */
size_t spd_workspace_bytes_rows(int64_t n_dm, int64_t n_t, int nmax);
spd_status spd_stats_rows(const float *d_x, int64_t n_dm, int64_t n_t, int64_t row_stride, int nmax_for_sigma,
                          spd_stats_t *d_stats_rows, void *d_ws, size_t ws_bytes, void *stream);
spd_status spd_boxcar_snr_rows(const float *d_x, int64_t n_dm, int64_t n_t, int64_t row_stride,
                               const spd_stats_t *d_stats_rows, int nmax, spd_sigma_mode mode,
                               float *d_snr, uint16_t *d_width, void *d_ws, size_t ws_bytes, void *stream);
spd_status spd_search_fused_rows(const float *d_x, int64_t n_dm, int64_t n_t, int64_t row_stride,
                                 const spd_stats_t *d_stats_rows, int nmax, spd_sigma_mode mode, float threshold,
                                 spd_candidate_t *d_out, uint64_t capacity, unsigned long long *d_count,
                                 void *d_ws, size_t ws_bytes, void *stream);

/* spd_stats_rows for callers that cannot obtain device memory of their own.
 * Who that is: a detection stage running inside somebody else's real-time pipeline.  The host framework owns the card: it
 * has split the whole of device memory into its own pools at start-up, passes each stage the device buffers it reads and
 * writes, and does not let a stage call cudaMalloc (the memory is already spoken for, and an allocation makes the device
 * wait, which would stall the other stages' streams mid-observation).  Such a caller has its input and its result buffer,
 * but nowhere to put the workspace spd_stats_rows needs.  Here the workspace is a fixed array inside libspd.so instead.
 *
 * Same arguments, kernels and results as spd_stats_rows (bit for bit), minus d_ws / ws_bytes.  d_x and d_stats_rows are
 * still the caller's.  The call allocates nothing: no cudaMalloc / cudaFree and no library routine that allocates.
 * Limit: n_dm <= SPD_NOALLOC_MAX_ROWS (8192; spd_stats_rows_noalloc_max_rows() returns it).  More rows than that return
 * SPD_ERR_NOALLOC_LIMIT before anything is launched: split the rows over several calls, one after the other on one stream.
 * Cost: the array is 3 MiB (8192 rows x 8 partials x 2 x 24 bytes) of device memory on EVERY GPU that loads the library,
 * held until the process exits, also by programs that never call this.
 * First call on a device: it looks up the array's device address (cudaGetSymbolAddress) and remembers it, with that device
 * current; make that first call during start-up, before any stream capture begins.  Later calls only enqueue kernels.
 * Shared state: all calls on one device use the same array.  It still holds the previous call's partials; nothing needs
 * clearing, because a call overwrites every slot it later reads.  Two calls that can overlap on the GPU (different streams
 * without an ordering between them, or two host threads on different streams) race on the array and give wrong statistics:
 * keep calls on one stream, or order them with events.  This is the one entry point of the library that keeps state. */
#define SPD_NOALLOC_MAX_ROWS 8192
int64_t spd_stats_rows_noalloc_max_rows(void);
spd_status spd_stats_rows_noalloc(const float *d_x, int64_t n_dm, int64_t n_t, int64_t row_stride, int nmax_for_sigma,
                                  spd_stats_t *d_stats_rows, void *stream);

/* Decimation in time + boxcar for wide filters (section 3: "a combination of boxcar filtering with the
 * decimation in time of the input data"; the paper names the route, the algorithm is reading A20 of DESIGN.md).
 * An APPROXIMATION of spd_boxcar_snr with nmax = w0 * 2^(levels-1): the width grid gets coarser with width
 * (PAPER.md:21, :69 warn about the sensitivity this costs: at most 1 - sqrt(0.9) = 5.1 % for w0 = 16).
 *   level 0: every width 1..w0 at every sample (exactly spd_boxcar_snr with nmax = w0 in the SQRT mode; in the LINEAR
 *            modes sigma_N is that of the whole search, Nmax = w0 * 2^(levels-1), so it equals the widths 1..w0 of
 *            spd_boxcar_snr with nmax = Nmax);
 *   level l: x_l[i] = x_{l-1}[2i] + x_{l-1}[2i+1] (n_l = n_t >> l samples per row), widths w' = w0/2+1..w0 of x_l at every
 *            decimated sample i: effective width N = w' 2^l, start sample t = i 2^l,
 *            SNR = (B - N mu) / sigma_N with sigma_N of the exhaustive search of the same nmax (eq. 4 / eq. 5 / anchored).
 * The kernels form the level series from the mean-subtracted samples (x_1[i] = (x[2i] - mu) + (x[2i+1] - mu), in fp32), so a
 * baseline far above the noise (|mu| = 1e3 sigma and more) costs the higher levels no precision.
 * Planes are packed per row: level l occupies elements [spd_decimated_level_offset(n_t, l), + n_l) of a row of
 * plane_stride elements (>= spd_decimated_level_offset(n_t, levels), a multiple of 8).  d_width holds the EFFECTIVE width
 * N; a position where none of the level's widths fits has snr = -inf, width = 0.
 * Requires w0 in {16, 32}, 1 <= levels <= 8, w0 <= n_t, w0 * 2^(levels-1) <= 4096.  d_ws: >= spd_decimated_workspace_bytes()
 * bytes, 256-byte aligned (it holds the decimated series of two levels at a time).  LINEAR modes need d_stats measured
 * with nmax_for_sigma = w0 * 2^(levels-1). */
int64_t spd_decimated_level_offset(int64_t n_t, int level);
size_t spd_decimated_workspace_bytes(int64_t n_dm, int64_t n_t, int w0, int levels);
spd_status spd_boxcar_snr_decimated(const float *d_x, int64_t n_dm, int64_t n_t, int64_t row_stride,
                                    const spd_stats_t *d_stats, int w0, int levels, spd_sigma_mode mode,
                                    float *d_snr, uint16_t *d_width, int64_t plane_stride,
                                    void *d_ws, size_t ws_bytes, void *stream);

/* Candidate selection over the packed planes of spd_boxcar_snr_decimated: one list for all levels,
 * record.t = start sample in the ORIGINAL series (i 2^l), record.width = effective width.  A pulse is usually reported by
 * several levels (the list is unordered and not clustered).  *d_count / capacity follow spd_candidates. */
spd_status spd_candidates_decimated(const float *d_snr, const uint16_t *d_width, int64_t n_dm, int64_t n_t, int64_t plane_stride,
                                    int levels, float threshold, spd_candidate_t *d_out, uint64_t capacity,
                                    unsigned long long *d_count, void *stream);

/* The decimated search with the threshold applied in the level kernels (steps 2-4 fused, as spd_search_fused is for the
 * exhaustive search): the level planes are never written.  Same records as spd_boxcar_snr_decimated +
 * spd_candidates_decimated -- (dm, t, snr) bit for bit; the width of a hit is found by replaying its running sums, so it is
 * the exact smallest arg-max among the level's widths and can differ from the plane path's only inside near-ties.
 * Arguments, workspace and the LINEAR-mode requirement follow spd_boxcar_snr_decimated; *d_count / capacity follow
 * spd_candidates; a LINEAR mode fed stats of another Nmax sets *d_count = UINT64_MAX, as spd_search_fused does. */
spd_status spd_search_fused_decimated(const float *d_x, int64_t n_dm, int64_t n_t, int64_t row_stride,
                                      const spd_stats_t *d_stats, int w0, int levels, spd_sigma_mode mode, float threshold,
                                      spd_candidate_t *d_out, uint64_t capacity, unsigned long long *d_count,
                                      void *d_ws, size_t ws_bytes, void *stream);

/* Device bytes spd_search_host needs in d_arena for this shape and capacity. */
size_t spd_search_host_arena_bytes(int64_t n_dm, int64_t n_t, int nmax, uint64_t capacity);

/* The whole path from HOST buffers: copies h_x (row_stride = n_t) to the device, runs spd_stats and
 * spd_search_fused (the list is the product; the planes are not materialised), and copies the
 * statistics, the hit count and the first min(count, capacity) records back.  h_x / h_out / h_count /
 * h_stats are HOST pointers (pinned memory makes the copies asynchronous); d_arena is a caller-owned DEVICE
 * buffer of >= spd_search_host_arena_bytes(), 256-byte aligned.  This call SYNCHRONISES `stream` before it returns
 * (once when count <= 4096: the first min(capacity, 4096) slots of h_out are copied together with the count, so h_out
 * entries past the count, up to that many, hold unspecified bytes afterwards; a longer list takes a second copy). */
spd_status spd_search_host(const float *h_x, int64_t n_dm, int64_t n_t, int nmax, spd_sigma_mode mode,
                           float threshold, spd_candidate_t *h_out, uint64_t capacity,
                           unsigned long long *h_count, spd_stats_t *h_stats,
                           void *d_arena, size_t arena_bytes, void *stream);

/* spd_search_host with the decimated search (the real-time route for wide filters): copies h_x to the device,
 * runs spd_stats (with sigma_Nmax of Nmax = w0 * 2^(levels-1) in the LINEAR modes) and spd_search_fused_decimated, and copies
 * the statistics, the hit count and the records back.  Arguments, the h_out convention and the synchronisation follow
 * spd_search_host; w0 / levels follow spd_boxcar_snr_decimated; d_arena: >= spd_search_host_decimated_arena_bytes() bytes
 * (0 = invalid arguments), 256-byte aligned. */
size_t spd_search_host_decimated_arena_bytes(int64_t n_dm, int64_t n_t, int w0, int levels, uint64_t capacity);
spd_status spd_search_host_decimated(const float *h_x, int64_t n_dm, int64_t n_t, int w0, int levels, spd_sigma_mode mode,
                                     float threshold, spd_candidate_t *h_out, uint64_t capacity,
                                     unsigned long long *h_count, spd_stats_t *h_stats,
                                     void *d_arena, size_t arena_bytes, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* SPD_H */
