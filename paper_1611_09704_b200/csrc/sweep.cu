// sweep.cu -- steps 2-4a: boxcars of every width, SNR, max / arg-max over width, one kernel
// (section 2.3, Algorithm 1; readings A5-A9 of DESIGN.md).
//
//   B_N(t) = sum_{k<N} x[t+k];  SNR_N(t) = (B_N(t) - N mu) / sigma_N;  snr[t] = max_N, width[t] = smallest arg-max.
//
// Design (sm_100a; this is NOT the paper's one-thread-X-samples loop):
//  * y = x - mu is formed once per sample while the tile is staged into shared memory (fp64 subtract, fp32
//    result), so the inner loop is B += y; s = B * r_N with r_N = 1/sigma_N from a table: no divide, no sqrt.
//  * One CTA owns 2048 consecutive samples of one row, as two sub-tiles A = [T0, T0+1024), B = [T0+1024, T0+2048).
//    Shared memory holds them INTERLEAVED as float2 Z[i] = (yA[i], yB[i]) so that one packed FADD2 / FMUL2
//    (Blackwell packed fp32) advances one running sum of each sub-tile: the FMA pipe sees 2 lane-ops per
//    (sample, width) pair -- the arithmetic floor -- for ONE issue slot per pair.
//  * Each thread owns 8 consecutive samples of each sub-tile and keeps a sliding window of 8 float2 in registers
//    (the width loop is unrolled by 8, so the rotation is register renaming): one LDS.64 per width step.
//  * Samples past the row end are staged as -inf: a running sum that has touched one is -inf for every wider
//    width, so "only widths that fit" (reading A9) needs no masking in the loop.
//  * arg-max is deferred: per block of 8 widths only the block maximum is formed (3-input FMNMX), one
//    compare/select per block records the winning block and the running sum at its start; after the loop the
//    winning block alone is re-summed in the same order (bit-identical) to find the smallest width attaining
//    the maximum.  Blocks ascend and every comparison is a strict '>' , so ties keep the smallest width (A7).
//
// Roofline: 10 B/sample of HBM traffic (4 read + 4 snr + 2 width) against 2*Nmax fp32 lane-ops per sample on the
// FMA pipe: FP32-pipe-bound for Nmax > ~28.
#include "spd_common.cuh"

namespace spd {

constexpr int SW_THREADS = 128;
constexpr int SW_R       = 8;                        // samples per thread per sub-tile
constexpr int SW_SUB     = SW_THREADS * SW_R;        // 1024
constexpr int SW_TILE    = 2 * SW_SUB;               // 2048 samples per CTA

__host__ __device__ inline int zpad(int i) { return i + (i >> 3); }          // one pad float2 per 8: lane stride 72 B
__host__ __device__ inline int sw_len(int nmax) { return SW_SUB + round_up(nmax, 8) + 16; }
__host__ __device__ inline int sw_rt_len(int nmax) { return round_up(nmax, 8) + 8; }

size_t sweep_table_bytes(int nmax) { return (size_t)sw_rt_len(nmax) * sizeof(float); }

__device__ __forceinline__ float fmax3(float a, float b, float c) { return fmaxf(fmaxf(a, b), c); }

// r_w = 1/sigma_w for w = 1..nmax: eq. 4, eq. 5 as printed, or the anchored variant.
// fp64 throughout, rounded once to fp32.  LINEAR modes fed stats measured for another Nmax write NaN.
__global__ void sigma_table_kernel(const spd_stats_t *__restrict__ st, int nmax, int mode, float *__restrict__ table)
{
    const double sigma = st->sigma, snm = st->sigma_nmax;
    const bool bad = (mode != SPD_SIGMA_SQRT) && (st->nmax_of_sigma != nmax);
    for (int w = 1 + blockIdx.x * blockDim.x + threadIdx.x; w <= sw_rt_len(nmax); w += gridDim.x * blockDim.x) {
        float r = 0.0f;
        if (w <= nmax) {
            double s = sqrt((double)w) * sigma;
            if (mode == SPD_SIGMA_LINEAR && nmax > 1) s += (double)(w - 1) * snm / (double)(nmax - 1);
            if (mode == SPD_SIGMA_LINEAR_ANCHORED && nmax > 1)
                s += (double)(w - 1) * (snm - sqrt((double)nmax) * sigma) / (double)(nmax - 1);
            r = bad ? __int_as_float(0x7fc00000) : (float)(1.0 / s);
        }
        table[w - 1] = r;
    }
}

cudaError_t launch_sigma_table(const spd_stats_t *d_stats, int nmax, int mode, float *d_table, cudaStream_t s)
{
    int n = sw_rt_len(nmax);
    sigma_table_kernel<<<(n + 255) / 256, 256, 0, s>>>(d_stats, nmax, mode, d_table);
    return cudaGetLastError();
}

template <bool FUSED>
__global__ void __launch_bounds__(SW_THREADS, 3)
boxcar_snr_sweep(const float *__restrict__ x, int64_t n_t, int64_t row_stride, int tiles_per_row,
                 const spd_stats_t *__restrict__ st, const float *__restrict__ table, int nmax,
                 float *__restrict__ snr, uint16_t *__restrict__ width,
                 float threshold, spd_candidate_t *__restrict__ cand, unsigned long long capacity,
                 unsigned long long *__restrict__ count)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int L = sw_len(nmax);
    float2 *Z  = reinterpret_cast<float2 *>(smem_raw);
    float2 *rt = Z + ((zpad(L) + 1) & ~1);

    const int tid = threadIdx.x;
    const int64_t row = blockIdx.x / tiles_per_row;
    const int64_t T0 = (int64_t)(blockIdx.x - row * tiles_per_row) * SW_TILE;
    const float *rowp = x + row * row_stride;
    const double mu = st->mean;
    const float NINF = __int_as_float(0xff800000);

    // ---- stage: y = x - mu, two sub-tiles interleaved; past the row end -> -inf -------------------------------
    {
        const bool vec = ((reinterpret_cast<uintptr_t>(rowp) & 15) == 0);
        for (int p = tid; p < L / 4; p += SW_THREADS) {
            const int i = 4 * p;
            float a[4], b[4];
            const int64_t pa = T0 + i, pb = T0 + SW_SUB + i;
            if (vec && pa + 3 < n_t) { float4 v = __ldg(reinterpret_cast<const float4 *>(rowp + pa)); a[0] = v.x; a[1] = v.y; a[2] = v.z; a[3] = v.w; }
            else { for (int k = 0; k < 4; ++k) a[k] = (pa + k < n_t) ? __ldg(rowp + pa + k) : NINF; }
            if (vec && pb + 3 < n_t) { float4 v = __ldg(reinterpret_cast<const float4 *>(rowp + pb)); b[0] = v.x; b[1] = v.y; b[2] = v.z; b[3] = v.w; }
            else { for (int k = 0; k < 4; ++k) b[k] = (pb + k < n_t) ? __ldg(rowp + pb + k) : NINF; }
#pragma unroll
            for (int k = 0; k < 4; ++k)
                Z[zpad(i + k)] = make_float2((float)((double)a[k] - mu), (float)((double)b[k] - mu));
        }
        for (int w = tid; w < sw_rt_len(nmax); w += SW_THREADS) { float r = __ldg(table + w); rt[w] = make_float2(r, r); }
    }
    __syncthreads();

    // ---- per-thread state --------------------------------------------------------------------------------------
    float2 B[SW_R], W[SW_R], best[SW_R], snap[SW_R];
    int blkx[SW_R], blky[SW_R];
#pragma unroll
    for (int j = 0; j < SW_R; ++j) {
        B[j] = make_float2(0.f, 0.f);
        W[j] = Z[9 * tid + j];                               // zpad(8 tid + j) = 9 tid + j
        best[j] = make_float2(NINF, NINF);
        snap[j] = make_float2(0.f, 0.f);
        blkx[j] = 0; blky[j] = 0;
    }
    const int nblk = nmax >> 3;

    // ---- main loop: one iteration = one block of 8 widths ------------------------------------------------------
    for (int kb = 0; kb < nblk; ++kb) {
        const float2 *zp = Z + 9 * (tid + kb + 1);           // zpad(8 tid + 8 kb + 8 + u) = 9 (tid + kb + 1) + u
        const float2 *rp = rt + 8 * kb;
        float2 B0[SW_R], m[SW_R];
#pragma unroll
        for (int j = 0; j < SW_R; ++j) B0[j] = B[j];
#pragma unroll
        for (int u = 0; u < 8; u += 2) {
            const float4 rr = *reinterpret_cast<const float4 *>(rp + u);
            const float2 r0 = make_float2(rr.x, rr.y), r1 = make_float2(rr.z, rr.w);
            float2 s0[SW_R], s1[SW_R];
#pragma unroll
            for (int j = 0; j < SW_R; ++j) { B[j] = __fadd2_rn(B[j], W[(j + u) & 7]); s0[j] = __fmul2_rn(B[j], r0); }
            W[u] = zp[u];
#pragma unroll
            for (int j = 0; j < SW_R; ++j) { B[j] = __fadd2_rn(B[j], W[(j + u + 1) & 7]); s1[j] = __fmul2_rn(B[j], r1); }
            W[u + 1] = zp[u + 1];
#pragma unroll
            for (int j = 0; j < SW_R; ++j) {
                if (u == 0) { m[j].x = fmaxf(s0[j].x, s1[j].x); m[j].y = fmaxf(s0[j].y, s1[j].y); }
                else        { m[j].x = fmax3(m[j].x, s0[j].x, s1[j].x); m[j].y = fmax3(m[j].y, s0[j].y, s1[j].y); }
            }
        }
#pragma unroll
        for (int j = 0; j < SW_R; ++j) {
            const bool px = m[j].x > best[j].x, py = m[j].y > best[j].y;
            best[j].x = px ? m[j].x : best[j].x;  snap[j].x = px ? B0[j].x : snap[j].x;  blkx[j] = px ? kb : blkx[j];
            best[j].y = py ? m[j].y : best[j].y;  snap[j].y = py ? B0[j].y : snap[j].y;  blky[j] = py ? kb : blky[j];
        }
    }

    // ---- re-sum the winning block (same order, same roundings) to find the smallest width attaining best --------
    int wx[SW_R], wy[SW_R];
#pragma unroll
    for (int j = 0; j < SW_R; ++j) {
        wx[j] = 1; wy[j] = 1;
        if (nblk > 0) {
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int kb = h ? blky[j] : blkx[j];
                const float bst = h ? best[j].y : best[j].x;
                float b = h ? snap[j].y : snap[j].x;
                const float *zf = reinterpret_cast<const float *>(Z + 9 * (tid + kb)) + h;
                const float *rf = reinterpret_cast<const float *>(rt + 8 * kb);
                float s[8];
#pragma unroll
                for (int g = 0; g < 8; ++g) { const int c = j + g; b += zf[2 * (c + (c >> 3))]; s[g] = b * rf[2 * g]; }
                int w = 0;
#pragma unroll
                for (int g = 7; g >= 0; --g) w = (s[g] == bst) ? g : w;
                if (h) wy[j] = 8 * kb + w + 1; else wx[j] = 8 * kb + w + 1;
            }
        }
    }

    // ---- tail widths (nmax not a multiple of 8): plain per-width tracking, wider widths so strict '>' still right
    const int rem = nmax & 7;
    if (rem) {
        const float2 *zp = Z + 9 * (tid + nblk + 1);
        for (int u = 0; u < rem; ++u) {
            const float2 r = rt[8 * nblk + u];
            const int wv = 8 * nblk + u + 1;
#pragma unroll
            for (int j = 0; j < SW_R; ++j) {
                B[j] = __fadd2_rn(B[j], W[j]);
                const float2 s = __fmul2_rn(B[j], r);
                if (s.x > best[j].x) { best[j].x = s.x; wx[j] = wv; }
                if (s.y > best[j].y) { best[j].y = s.y; wy[j] = wv; }
            }
#pragma unroll
            for (int j = 0; j < SW_R - 1; ++j) W[j] = W[j + 1];      // rem < 8 steps: a plain shift is fine here
            W[SW_R - 1] = zp[u];
        }
    }

    // a NaN reciprocal table (LINEAR mode fed stats of another Nmax) must surface: fmaxf drops NaN operands
    if (rt[0].x != rt[0].x) {
#pragma unroll
        for (int j = 0; j < SW_R; ++j) best[j] = make_float2(rt[0].x, rt[0].x);
    }

    // ---- results --------------------------------------------------------------------------------------------------
    const int64_t ta = T0 + SW_R * tid, tb = ta + SW_SUB;
    if (!FUSED) {
        float *oa = snr + row * row_stride + ta, *ob = snr + row * row_stride + tb;
        const bool v4 = ((reinterpret_cast<uintptr_t>(snr + row * row_stride) & 15) == 0);
        if (v4 && ta + 7 < n_t) {
            reinterpret_cast<float4 *>(oa)[0] = make_float4(best[0].x, best[1].x, best[2].x, best[3].x);
            reinterpret_cast<float4 *>(oa)[1] = make_float4(best[4].x, best[5].x, best[6].x, best[7].x);
        } else {
#pragma unroll
            for (int j = 0; j < SW_R; ++j) if (ta + j < n_t) oa[j] = best[j].x;
        }
        if (v4 && tb + 7 < n_t) {
            reinterpret_cast<float4 *>(ob)[0] = make_float4(best[0].y, best[1].y, best[2].y, best[3].y);
            reinterpret_cast<float4 *>(ob)[1] = make_float4(best[4].y, best[5].y, best[6].y, best[7].y);
        } else {
#pragma unroll
            for (int j = 0; j < SW_R; ++j) if (tb + j < n_t) ob[j] = best[j].y;
        }
        if (width) {
            uint16_t *wa = width + row * row_stride + ta, *wb = width + row * row_stride + tb;
            const bool w8 = ((reinterpret_cast<uintptr_t>(width + row * row_stride) & 15) == 0);
            if (w8 && ta + 7 < n_t)
                *reinterpret_cast<uint4 *>(wa) = make_uint4(wx[0] | (wx[1] << 16), wx[2] | (wx[3] << 16), wx[4] | (wx[5] << 16), wx[6] | (wx[7] << 16));
            else {
#pragma unroll
                for (int j = 0; j < SW_R; ++j) if (ta + j < n_t) wa[j] = (uint16_t)wx[j];
            }
            if (w8 && tb + 7 < n_t)
                *reinterpret_cast<uint4 *>(wb) = make_uint4(wy[0] | (wy[1] << 16), wy[2] | (wy[3] << 16), wy[4] | (wy[5] << 16), wy[6] | (wy[7] << 16));
            else {
#pragma unroll
                for (int j = 0; j < SW_R; ++j) if (tb + j < n_t) wb[j] = (uint16_t)wy[j];
            }
        }
    } else {
        // threshold in the same kernel: planes are never written
        bool any = false;
#pragma unroll
        for (int j = 0; j < SW_R; ++j) any |= (best[j].x >= threshold && ta + j < n_t) || (best[j].y >= threshold && tb + j < n_t);
        if (__any_sync(0xffffffffu, any)) {
#pragma unroll
            for (int j = 0; j < SW_R; ++j) {
                append_candidate(best[j].x >= threshold && ta + j < n_t, (uint32_t)row, (uint32_t)(ta + j), best[j].x, (uint32_t)wx[j], cand, capacity, count);
                append_candidate(best[j].y >= threshold && tb + j < n_t, (uint32_t)row, (uint32_t)(tb + j), best[j].y, (uint32_t)wy[j], cand, capacity, count);
            }
        }
    }
}

cudaError_t launch_sweep(const float *x, int64_t n_dm, int64_t n_t, int64_t row_stride, const spd_stats_t *d_stats,
                         const float *d_table, int nmax, float *snr, uint16_t *width,
                         bool fused, float threshold, spd_candidate_t *out, unsigned long long capacity,
                         unsigned long long *d_count, cudaStream_t s)
{
    const int tpr = (int)((n_t + SW_TILE - 1) / SW_TILE);
    const int64_t blocks = n_dm * (int64_t)tpr;
    if (blocks > 2147483647LL) return cudaErrorInvalidConfiguration;
    const size_t smem = (size_t)((zpad(sw_len(nmax)) + 1) & ~1) * sizeof(float2) + (size_t)sw_rt_len(nmax) * sizeof(float2);
    cudaError_t e;
    if (fused) {
        e = cudaFuncSetAttribute(boxcar_snr_sweep<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        boxcar_snr_sweep<true><<<(unsigned)blocks, SW_THREADS, smem, s>>>(x, n_t, row_stride, tpr, d_stats, d_table, nmax,
                                                                         nullptr, nullptr, threshold, out, capacity, d_count);
    } else {
        e = cudaFuncSetAttribute(boxcar_snr_sweep<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        boxcar_snr_sweep<false><<<(unsigned)blocks, SW_THREADS, smem, s>>>(x, n_t, row_stride, tpr, d_stats, d_table, nmax,
                                                                          snr, width, 0.0f, nullptr, 0, nullptr);
    }
    return cudaGetLastError();
}

}  // namespace spd
