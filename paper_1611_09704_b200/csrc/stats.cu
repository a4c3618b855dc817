// stats.cu -- step 1 of the path: mean and standard deviation (section 2.1).
//
// Kernel 1 (stats_partial): the array is cut into equal chunks of 4096 samples; every thread runs the
// streaming update eq. 1 over a fixed run of 16 samples (division-free: 1/(j(j-1)) are compile-time
// constants), the 32 runs of a warp are merged pairwise with eq. 2 through shuffles, and the warp's
// 512-sample partial is merged (eq. 2, fp64) into a per-warp accumulator.  Each CTA writes one
// (m, T, S) partial.  Kernel 2 (stats_finalize) merges the partials with eq. 2 in index order (fp64,
// fixed order => bit-reproducible) and writes mu = T/n, sigma = sqrt(S/n).
//
// Precision (reading A4): fp32 inside a warp-chunk (<= 512 samples), fp64 above it.  All
// samples are shifted by K = x[0][0] before they enter eq. 1 (eq. 1/2 are applied to x - K; S is
// shift-invariant and T is un-shifted at the end), which keeps fp32 accurate when |mu| >> sigma.
//
// Roofline: pure HBM stream, 4 B/sample read.
#include "spd_common.cuh"

namespace spd {

constexpr int ST_THREADS = 256;
constexpr int ST_RUN     = 16;                       // samples per thread-run (4 x float4)
constexpr int ST_CHUNK   = ST_THREADS * ST_RUN;      // 4096 samples
constexpr int ST_GRID    = 148 * 8;                  // persistent CTAs (<= MAX_PARTIALS)

__device__ __forceinline__ float4 ldg_stream4(const float *p)
{
    float4 v;
    asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];"
                 : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
    return v;
}

// eq. 1 for the j-th sample of a run, j a compile-time constant >= 2:
//   T_j = T_{j-1} + x_j ;  S_j = S_{j-1} + (j x_j - T_j)^2 / (j (j-1))
template <int J>
__device__ __forceinline__ void chan_push(float &T, float &S, float x)
{
    T += x;
    float d = fmaf((float)J, x, -T);
    S = fmaf(d * d, 1.0f / (float)(J * (J - 1)), S);
}

// eq. 2 for two partials of EQUAL size m: S = S1 + S2 + (T1 - T2)^2 / (2m)
__device__ __forceinline__ void merge_equal(float &T, float &S, float T2, float S2, float inv_2m)
{
    float d = T - T2;
    S = fmaf(d * d, inv_2m, S + S2);
    T += T2;
}

__global__ void __launch_bounds__(ST_THREADS)
stats_partial(const float *__restrict__ x, int64_t n_rows, int64_t n_t, int64_t row_stride, Tri *__restrict__ partials)
{
    __shared__ Tri warp_acc[ST_THREADS / 32];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const float K = __ldg(x);                                  // shift (see header)
    const int64_t cpr = (n_t + ST_CHUNK - 1) / ST_CHUNK;       // chunks per row
    const int64_t total = n_rows * cpr;
    Tri acc = {0.0, 0.0, 0.0};                                 // lane 0 of each warp owns it

    for (int64_t c = blockIdx.x; c < total; c += gridDim.x) {
        const int64_t row = c / cpr, off = (c - row * cpr) * ST_CHUNK;
        const float *base = x + row * row_stride + off;
        const bool full = (off + ST_CHUNK <= n_t) && ((reinterpret_cast<uintptr_t>(base) & 15) == 0);
        if (full) {
            float4 v[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) v[k] = ldg_stream4(base + (k * ST_THREADS + tid) * 4);
            float T = v[0].x - K, S = 0.0f;
            chan_push<2>(T, S, v[0].y - K);  chan_push<3>(T, S, v[0].z - K);  chan_push<4>(T, S, v[0].w - K);
            chan_push<5>(T, S, v[1].x - K);  chan_push<6>(T, S, v[1].y - K);  chan_push<7>(T, S, v[1].z - K);
            chan_push<8>(T, S, v[1].w - K);  chan_push<9>(T, S, v[2].x - K);  chan_push<10>(T, S, v[2].y - K);
            chan_push<11>(T, S, v[2].z - K); chan_push<12>(T, S, v[2].w - K); chan_push<13>(T, S, v[3].x - K);
            chan_push<14>(T, S, v[3].y - K); chan_push<15>(T, S, v[3].z - K); chan_push<16>(T, S, v[3].w - K);
#pragma unroll
            for (int lvl = 0; lvl < 5; ++lvl) {                // 16 -> 512 samples, equal sizes at each level
                float T2 = __shfl_xor_sync(0xffffffffu, T, 1 << lvl);
                float S2 = __shfl_xor_sync(0xffffffffu, S, 1 << lvl);
                merge_equal(T, S, T2, S2, 1.0f / (float)(2 * (ST_RUN << lvl)));
            }
            if (lane == 0) { Tri w = {512.0, (double)T, (double)S}; tri_merge(acc, w); }
        } else {
            // ragged / unaligned chunk: eq. 1 with a run-time j, eq. 2 merges in fp64
            Tri t = {0.0, 0.0, 0.0};
            float T = 0.0f, S = 0.0f; int j = 0;
            for (int k = 0; k < ST_RUN; ++k) {
                int64_t p = off + (int64_t)((k >> 2) * ST_THREADS + tid) * 4 + (k & 3);
                if (p < n_t) {
                    float xv = __ldg(x + row * row_stride + p) - K;
                    ++j;
                    if (j == 1) { T = xv; S = 0.0f; }
                    else { T += xv; float d = fmaf((float)j, xv, -T); S += d * d / (float)(j * (j - 1)); }
                }
            }
            t.m = (double)j; t.T = (double)T; t.S = (double)S;
#pragma unroll
            for (int lvl = 0; lvl < 5; ++lvl) {
                Tri o;
                o.m = __shfl_xor_sync(0xffffffffu, t.m, 1 << lvl);
                o.T = __shfl_xor_sync(0xffffffffu, t.T, 1 << lvl);
                o.S = __shfl_xor_sync(0xffffffffu, t.S, 1 << lvl);
                if ((lane >> lvl) & 1) { Tri a = o; tri_merge(a, t); t = a; } else tri_merge(t, o);
            }
            if (lane == 0) tri_merge(acc, t);
        }
    }
    if (lane == 0) warp_acc[wid] = acc;
    __syncthreads();
    if (tid == 0) {
        Tri a = warp_acc[0];
        for (int w = 1; w < ST_THREADS / 32; ++w) tri_merge(a, warp_acc[w]);
        partials[blockIdx.x] = a;
    }
}

// ---- sigma_Nmax: population std of the Nmax-sample boxcar SUMS over every full window (reading A11) ----
// One tile = 4096 consecutive windows of one row (+ nmax-1 halo samples) staged in shared memory, together with its
// tile-local fp64 prefix sums P (block scan).  Each thread owns 16 consecutive windows: the first sum is
// P[t+nmax] - P[t], the next 15 slide (+x[t+nmax] - x[t], fp64), the sums go through eq. 1 (fp64) and the warp's runs
// are merged with eq. 2.
constexpr int SB_WIN = 16;
constexpr int SB_TILE = ST_THREADS * SB_WIN;
__host__ __device__ __forceinline__ int sb_pad(int i) { return i + (i >> 4); }   // lane stride 17 words: conflict-free

__global__ void __launch_bounds__(ST_THREADS)
stats_boxcar_partial(const float *__restrict__ x, int64_t n_dm, int64_t n_t, int64_t row_stride, int nmax,
                     Tri *__restrict__ partials)
{
    extern __shared__ __align__(16) unsigned char sb_smem[];
    __shared__ Tri warp_acc[ST_THREADS / 32];
    __shared__ double wtot[ST_THREADS / 32];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    double *Pd = reinterpret_cast<double *>(sb_smem);                              // [span + 1] prefix sums
    float *xs = reinterpret_cast<float *>(Pd + (SB_TILE + nmax));                  // [sb_pad(span) + 1] samples
    const int64_t nwin = n_t - nmax + 1;
    const int64_t tpr = (nwin + SB_TILE - 1) / SB_TILE;
    const int64_t total = n_dm * tpr;
    const int span = SB_TILE + nmax - 1;
    const int seg = (span + ST_THREADS - 1) / ST_THREADS;
    Tri acc = {0.0, 0.0, 0.0};

    for (int64_t c = blockIdx.x; c < total; c += gridDim.x) {
        const int64_t row = c / tpr, t0 = (c - row * tpr) * SB_TILE;
        const float *rp = x + row * row_stride;
        __syncthreads();
        for (int i = tid; i < span; i += ST_THREADS) xs[sb_pad(i)] = (t0 + i < n_t) ? __ldg(rp + t0 + i) : 0.0f;
        __syncthreads();
        {   // P[i] = xs[0] + ... + xs[i-1] in fp64: per-thread segment sums, warp scan, cross-warp offsets
            const int lo = min(tid * seg, span), hi = min(lo + seg, span);
            double run = 0.0;
            for (int i = lo; i < hi; ++i) run += (double)xs[sb_pad(i)];
            double inc = run;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) { const double o = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += o; }
            if (lane == 31) wtot[wid] = inc;
            __syncthreads();
            double off = inc - run;
            for (int w = 0; w < wid; ++w) off += wtot[w];
            for (int i = lo; i < hi; ++i) { Pd[i] = off; off += (double)xs[sb_pad(i)]; }
            if (hi == span && lo < hi) Pd[span] = off;           // the one thread whose non-empty segment ends the tile
        }
        __syncthreads();
        const int w0 = tid * SB_WIN;
        Tri t = {0.0, 0.0, 0.0};
        if (t0 + w0 < nwin) {
            double B = Pd[w0 + nmax] - Pd[w0];
            t.m = 1.0; t.T = B; t.S = 0.0;
#pragma unroll
            for (int r = 1; r < SB_WIN; ++r) {
                if (t0 + w0 + r < nwin) {
                    B += (double)xs[sb_pad(w0 + r - 1 + nmax)] - (double)xs[sb_pad(w0 + r - 1)];
                    const double j = (double)(r + 1);
                    t.T += B;
                    double d = j * B - t.T;
                    t.S += d * d * (1.0 / (j * (j - 1.0)));
                    t.m = j;
                }
            }
        }
        if (__all_sync(0xffffffffu, t.m == (double)SB_WIN)) {
            // every run is full: eq. 2 for equal sizes m, S = S1 + S2 + (T1 - T2)^2 / (2m), with 1/(2m) a constant
            // per level (no fp64 division); the order of the two operands is that of the general path below
#pragma unroll
            for (int lvl = 0; lvl < 5; ++lvl) {
                const double T2 = __shfl_xor_sync(0xffffffffu, t.T, 1 << lvl);
                const double S2 = __shfl_xor_sync(0xffffffffu, t.S, 1 << lvl);
                const double d = t.T - T2;
                t.S = (t.S + S2) + d * d * (1.0 / (double)(2 * (SB_WIN << lvl)));
                t.T += T2;
            }
            t.m = (double)(32 * SB_WIN);
        } else {
#pragma unroll
            for (int lvl = 0; lvl < 5; ++lvl) {
                Tri o;
                o.m = __shfl_xor_sync(0xffffffffu, t.m, 1 << lvl);
                o.T = __shfl_xor_sync(0xffffffffu, t.T, 1 << lvl);
                o.S = __shfl_xor_sync(0xffffffffu, t.S, 1 << lvl);
                if ((lane >> lvl) & 1) { Tri a = o; tri_merge(a, t); t = a; } else tri_merge(t, o);
            }
        }
        if (lane == 0) tri_merge(acc, t);
    }
    if (lane == 0) warp_acc[wid] = acc;
    __syncthreads();
    if (tid == 0) {
        Tri a = warp_acc[0];
        for (int w = 1; w < ST_THREADS / 32; ++w) tri_merge(a, warp_acc[w]);
        partials[blockIdx.x] = a;
    }
}

// ---- kernel 2: merge the block partials (eq. 2, fp64, fixed order) and write the result -----------------
__device__ Tri fold_partials(const Tri *p, int count, Tri *sh)
{
    const int tid = threadIdx.x;
    const int per = (count + ST_THREADS - 1) / ST_THREADS;
    Tri a = {0.0, 0.0, 0.0};
    for (int i = tid * per; i < min(count, (tid + 1) * per); ++i) tri_merge(a, p[i]);
    sh[tid] = a;
    __syncthreads();
    for (int s = 1; s < ST_THREADS; s <<= 1) {                 // in-order binary tree over contiguous segments
        if ((tid & (2 * s - 1)) == 0) { Tri b = sh[tid + s]; tri_merge(sh[tid], b); }
        __syncthreads();
    }
    Tri r = sh[0];
    __syncthreads();
    return r;
}

__device__ __forceinline__ void fill_stats(spd_stats_t *out, const Tri &a, const Tri &b, int nmax_of_sigma)
{
    out->n = (uint64_t)a.m; out->T = a.T; out->S = a.S;
    out->mean = a.T / a.m;
    out->sigma = sqrt(a.S / a.m);
    out->n_b = (uint64_t)b.m; out->T_b = b.T; out->S_b = b.S;
    out->sigma_nmax = (nmax_of_sigma > 0 && b.m > 0.0) ? sqrt(b.S / b.m) : __longlong_as_double(0x7ff8000000000000LL);
    out->nmax_of_sigma = nmax_of_sigma; out->_pad = 0;
}

__global__ void __launch_bounds__(ST_THREADS)
stats_finalize(const float *__restrict__ x, const Tri *__restrict__ part_x, int count_x,
               const Tri *__restrict__ part_b, int count_b, int nmax_of_sigma, spd_stats_t *__restrict__ out)
{
    __shared__ Tri sh[ST_THREADS];
    Tri a = fold_partials(part_x, count_x, sh);
    Tri b = {0.0, 0.0, 0.0};
    if (count_b > 0) b = fold_partials(part_b, count_b, sh);
    if (threadIdx.x == 0) {
        a.T += a.m * (double)__ldg(x);                         // undo the shift K = x[0][0]
        fill_stats(out, a, b, nmax_of_sigma);
    }
}

// eq. 2 over whole results (the exchange step of a DM-row-sharded run), folded in index order
__global__ void stats_merge_kernel(const spd_stats_t *__restrict__ parts, int count, spd_stats_t *__restrict__ out)
{
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    Tri a = {0.0, 0.0, 0.0}, b = {0.0, 0.0, 0.0};
    int nm = parts[0].nmax_of_sigma;
    for (int i = 0; i < count; ++i) {
        Tri pa = {(double)parts[i].n, parts[i].T, parts[i].S}, pb = {(double)parts[i].n_b, parts[i].T_b, parts[i].S_b};
        tri_merge(a, pa); tri_merge(b, pb);
        if (parts[i].nmax_of_sigma != nm) nm = 0;
    }
    fill_stats(out, a, b, nm);
}

cudaError_t launch_stats(const float *x, int64_t n_dm, int64_t n_t, int64_t row_stride, int nmax_for_sigma,
                         spd_stats_t *d_stats, void *d_ws, cudaStream_t s)
{
    Tri *px = reinterpret_cast<Tri *>(d_ws), *pb = px + MAX_PARTIALS;
    int64_t rows = n_dm, cols = n_t, stride = row_stride;
    if (row_stride == n_t) { cols = n_dm * n_t; rows = 1; stride = cols; }     // contiguous: one long row
    int64_t chunks = rows * ((cols + ST_CHUNK - 1) / ST_CHUNK);
    int gx = (int)(chunks < ST_GRID ? chunks : ST_GRID);
    stats_partial<<<gx, ST_THREADS, 0, s>>>(x, rows, cols, stride, px);
    int gb = 0;
    if (nmax_for_sigma > 0) {
        int64_t nwin = n_t - nmax_for_sigma + 1;
        int64_t tiles = n_dm * ((nwin + SB_TILE - 1) / SB_TILE);
        gb = (int)(tiles < ST_GRID ? tiles : ST_GRID);
        size_t smem = (size_t)(SB_TILE + nmax_for_sigma) * sizeof(double) + (size_t)(sb_pad(SB_TILE + nmax_for_sigma) + 1) * sizeof(float);
        cudaError_t e = cudaFuncSetAttribute(stats_boxcar_partial, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        stats_boxcar_partial<<<gb, ST_THREADS, smem, s>>>(x, n_dm, n_t, row_stride, nmax_for_sigma, pb);
    }
    stats_finalize<<<1, ST_THREADS, 0, s>>>(x, px, gx, pb, gb, nmax_for_sigma, d_stats);
    return cudaGetLastError();
}

cudaError_t launch_stats_merge(const spd_stats_t *parts, int count, spd_stats_t *out, cudaStream_t s)
{
    stats_merge_kernel<<<1, 32, 0, s>>>(parts, count, out);
    return cudaGetLastError();
}

}  // namespace spd
