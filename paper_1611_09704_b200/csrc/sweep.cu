// sweep.cu -- steps 2-4a: boxcars of every width, SNR, max / arg-max over width, one kernel
// (section 2.3, Algorithm 1; readings A5-A9 of DESIGN.md).
//
//   B_N(t) = sum_{k<N} x[t+k];  SNR_N(t) = (B_N(t) - N mu) / sigma_N;  snr[t] = max_N, width[t] = smallest arg-max.
//
// Three kernels share one width loop (sweep8): boxcar_snr_sweep (planes, any nmax), boxcar_snr_sweep_narrow (planes,
// nmax <= 24) and boxcar_search_fused (threshold in the kernel, no planes).
//
// Design (sm_100a; this is NOT the paper's one-thread-X-samples loop):
//  * Persistent CTAs (one wave, grid = SMs x resident CTAs) walk the tiles; the raw samples of the NEXT tile are
//    prefetched with cp.async (LDGSTS, 16 B) into shared memory while the current tile is swept.
//  * y = x - mu is formed once per sample when the raw tile is converted into the working layout (two-term fp32
//    subtract, mu = mu_hi + mu_lo), so the inner loop is B += y; s = B * r_N with r_N = 1/sigma_N from a table.
//  * One tile = 2048 consecutive samples of one row, as two sub-tiles A = [T0, T0+1024), B = [T0+1024, T0+2048).
//    The working layout INTERLEAVES them, float2 Z[i] = (yA[i], yB[i]), so that one packed FADD2 / FMUL2
//    (Blackwell packed fp32) advances one running sum of each sub-tile.  Measured on B200: the
//    loop is bound by instruction dispatch and register-operand bandwidth, not by a pipe; a packed op costs two
//    dispatch clocks, like two scalar ones, but the packed mix is the fastest measured (about 10 % ahead of scalar),
//    and r_N enters FMUL2 as a scalar-broadcast operand (one register read less than a (r, r) pair: 4-8 % faster).
//  * Each thread owns 8 consecutive samples of each sub-tile and keeps a sliding window of 8 float2 in registers
//    (the width loop is unrolled by 8, so the rotation is register renaming): one LDS.64 per width step.
//  * Samples past the row end are staged as -inf: a running sum that has touched one is -inf for every wider
//    width, so "only widths that fit" (reading A9) needs no masking in the loop.  Widths nmax < w <= 8 ceil(nmax/8)
//    get a NaN reciprocal: FMNMX drops NaN operands, so they can never win and need no tail loop.
//  * arg-max of the general kernel is deferred: the running maximum is advanced with 3-input FMNMX only,
//    ping-ponging between two register sets so that the value before and after each block of 8 widths are both
//    live; one compare + one select per block then record the block that last raised it.  After the loop that block
//    alone is evaluated again from a tile-local prefix sum P kept in shared memory (B_w(t) = P[t+w] - P[t], no
//    dependency chain); the position inside the block rides in the 3 low mantissa bits of the 8 values (a larger tag
//    is a smaller width), so one maximum gives the width.  Blocks ascend with a strict '>', so exact ties keep the
//    smallest width (A7).  The SNR written is the running-sum value of the main loop; the re-evaluation only picks
//    the width and differs from the running sums by fp32 rounding and the 3 tag bits (~1e-6 relative), i.e. only
//    inside near-ties far below the 1e-3 tie tolerance.
//
// Roofline: 10 B/sample of HBM traffic (4 read + 4 snr + 2 width) against 3*Nmax fp32 lane-ops per sample (add,
// multiply, compare) at one warp instruction per sub-partition per clock: FP32-issue-bound for Nmax > ~20
// (DESIGN.md section 7).
#include "spd_common.cuh"

namespace spd {

constexpr int SW_R       = 8;                        // samples per thread per sub-tile
// CTA width NT (a template parameter of the kernels): sub-tile = 8 NT samples, tile = 16 NT samples of one row.
// 64 threads (tile 1024) for nmax <= SW_SMALL_CTA_NMAX: fewer warps wait on each block barrier; 128 threads (tile 2048)
// above, where the halo (nmax + 8 positions staged and scanned per tile) would weigh too much on a small tile.
constexpr int SW_SMALL_CTA_NMAX = 256;
constexpr int SW_NARROW_NMAX = 24;                   // nmax up to here takes the tagged-maximum kernel (measured crossover on B200: 24..28)

__host__ __device__ inline int zpad(int i) { return i + (i >> 3); }          // one pad float2 per 8: lane stride 72 B
__host__ __device__ inline int sw_nblk(int nmax) { return (nmax + 7) >> 3; }  // blocks of 8 widths
__host__ __device__ inline int sw_halo(int nmax) { return 8 * sw_nblk(nmax) + 8; }   // positions staged past a sub-tile
__host__ __device__ inline int sw_rt_len(int nmax) { return 8 * sw_nblk(nmax) + 8; } // reciprocal-table entries

size_t sweep_table_bytes(int nmax) { return (size_t)sw_rt_len(nmax) * sizeof(float); }

struct SweepSmem {           // byte offsets into dynamic shared memory (all 16-byte aligned)
    int z, raw, p2, scan, rtf, total;
    __host__ __device__ SweepSmem(int nmax, int nt)
    {
        const int H = sw_halo(nmax), R = sw_rt_len(nmax), SW_SUB = nt * SW_R, SW_TILE = 2 * SW_SUB;
        z = 0;                                                           // float2 Z[zpad(SUB + H)]
        raw = z + round_up((zpad(SW_SUB + H) + 1) * 8, 16);              // float raw[TILE + H]
        p2 = raw + round_up((SW_TILE + H) * 4, 16);                      // float2 P[zpad(SUB + H + 1)]: prefix sums
        scan = p2 + round_up((zpad(SW_SUB + H + 1) + 1) * 8, 16);        // float2 [2][4]: per-warp totals of the scan (double-buffered by part)
        rtf = scan + 64;                                                 // float r_w
        total = rtf + round_up(R * 4, 16);
    }
};

__device__ __forceinline__ float fmax3(float a, float b, float c) { return fmaxf(fmaxf(a, b), c); }

__device__ __forceinline__ void cp_async16(void *smem, const void *gmem)
{
    unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" :: "r"(s), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit_wait_all()
{
    asm volatile("cp.async.commit_group;\ncp.async.wait_group 0;" ::: "memory");
}

// r_w = 1/sigma_w for w = 1..nmax: eq. 4, eq. 5 as printed, or the anchored variant.
// fp64 throughout, rounded once to fp32.  LINEAR modes fed stats measured for another Nmax write NaN.
__global__ void sigma_table_kernel(const spd_stats_t *__restrict__ st, int nmax, int mode, float *__restrict__ table)
{
    const double sigma = st->sigma, snm = st->sigma_nmax;
    const bool bad = (mode != SPD_SIGMA_SQRT) && (st->nmax_of_sigma != nmax);
    for (int w = 1 + blockIdx.x * blockDim.x + threadIdx.x; w <= sw_rt_len(nmax); w += gridDim.x * blockDim.x) {
        float r = __int_as_float(0x7fc00000);      // widths past nmax (padding of the last block of 8) never win
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

// Position of a tile in the persistent walk: (row, tile-in-row), advanced by the grid size without 64-bit divisions
struct TilePos {
    int64_t row; int tr;
    __device__ __forceinline__ TilePos(unsigned first, int tiles_per_row) : row(first / (unsigned)tiles_per_row), tr((int)(first % (unsigned)tiles_per_row)) {}
    __device__ __forceinline__ TilePos next(unsigned step, int tiles_per_row) const
    {
        TilePos p = *this;
        unsigned t = (unsigned)p.tr + step;
        if (t >= (unsigned)tiles_per_row) { const unsigned q = t / (unsigned)tiles_per_row; p.row += q; t -= q * (unsigned)tiles_per_row; }
        p.tr = (int)t;
        return p;
    }
};

// ---- tile staging -------------------------------------------------------------------------------------------------
// An interior tile of a 16-byte aligned row is one contiguous run of global memory.  BULK: ONE thread issues a 1-D bulk
// copy (TMA: cp.async.bulk, completion counted in bytes on an mbarrier) and every thread waits on the barrier's phase;
// otherwise every thread issues 16-byte cp.async.  Measured on B200 (config-3 shape): the bulk copy is 2.7 % faster for
// the narrow kernel (Nmax 8, closest to the HBM roofline) and 1.4 % / 6 % SLOWER for the general and the fused kernel,
// so only the narrow kernel uses it.  Tiles that touch the row end, and rows that are not 16-byte aligned, are staged
// by all threads (cp.async 16 B where possible, scalar loads otherwise; samples past the row end become -inf).
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }

struct TileStager {
    unsigned long long *bar;
    unsigned phase;
    bool pending_bulk;

    __device__ __forceinline__ void init(unsigned long long *b, int tid)
    {
        bar = b; phase = 0; pending_bulk = false;
        if (tid == 0) {
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" :: "r"(smem_u32(b)) : "memory");
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
        __syncthreads();
    }

    template <int NT, bool BULK>
    __device__ __forceinline__ void stage(float *__restrict__ raw, const float *__restrict__ x, int64_t n_t, int64_t row_stride,
                                          const TilePos &pos_, int LRAW, int tid)
    {
        const float NINF = __int_as_float(0xff800000);
        const int64_t T0 = (int64_t)pos_.tr * (2 * NT * SW_R);
        const float *rowp = x + pos_.row * row_stride;
        const bool vec = ((reinterpret_cast<uintptr_t>(rowp) & 15) == 0);
        const bool interior = vec && (T0 + LRAW <= n_t);
        pending_bulk = BULK && interior;
        if (pending_bulk) {                                  // interior tile: one bulk copy
            if (tid == 0) {
                const unsigned bytes = (unsigned)LRAW * 4u;
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // earlier generic-proxy accesses of raw are ordered by the block barrier
                asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(smem_u32(bar)), "r"(bytes) : "memory");
                asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                             :: "r"(smem_u32(raw)), "l"(rowp + T0), "r"(bytes), "r"(smem_u32(bar)) : "memory");
            }
        } else if (interior) {                               // the same run, 16 bytes per thread and step
            const float *src = rowp + T0;
            for (int p = tid; p < LRAW / 4; p += NT) cp_async16(raw + 4 * p, src + 4 * p);
        } else {
            for (int p = tid; p < LRAW / 4; p += NT) {
                const int64_t pos = T0 + 4 * p;
                if (vec && pos + 3 < n_t) cp_async16(raw + 4 * p, rowp + pos);
                else {
#pragma unroll
                    for (int k = 0; k < 4; ++k) raw[4 * p + k] = (pos + k < n_t) ? __ldg(rowp + pos + k) : NINF;
                }
            }
        }
    }

    // the tile staged last has landed (for this thread; the block barrier that follows makes it so for all)
    __device__ __forceinline__ void wait()
    {
        if (pending_bulk) {
            unsigned ok;
            do {
                asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                             : "=r"(ok) : "r"(smem_u32(bar)), "r"(phase) : "memory");
            } while (!ok);
            phase ^= 1u;
        } else {
            cp_async_commit_wait_all();
        }
    }
};

// One block of 8 width steps: advance the 8 packed running sums, scale, fold into the running maxima.
// out[j] = max(in[j], the 8 SNRs of this block); `in` stays intact so that the caller can tell whether the block
// raised the maximum.  On entry W[v] = Z[8 tid + a0 + v] (a0 = width offset of the first step); on exit the window
// has moved by 8.  zp -> Z[8 (tid + kb + 1)] (the next 8 window elements), rp -> r_w of the block (a scalar operand:
// FMUL2 broadcasts one register to both halves, which costs one register read less than a (r_w, r_w) pair).
__device__ __forceinline__ void sweep8(float2 (&B)[SW_R], float2 (&W)[SW_R], const float2 (&in)[SW_R], float2 (&out)[SW_R],
                                       const float2 *__restrict__ zp, const float *__restrict__ rp)
{
#pragma unroll
    for (int u = 0; u < 8; u += 2) {
        const float2 rr = *reinterpret_cast<const float2 *>(rp + u);              // r_w of the two widths: scalar-broadcast operands of FMUL2
        const float2 r0 = make_float2(rr.x, rr.x), r1 = make_float2(rr.y, rr.y);
        const float2 n0 = zp[u], n1 = zp[u + 1];
#pragma unroll
        for (int j = 0; j < SW_R; ++j) {
            B[j] = __fadd2_rn(B[j], W[(j + u) & 7]);
            const float2 s0 = __fmul2_rn(B[j], r0);
            B[j] = __fadd2_rn(B[j], (j == SW_R - 1) ? n0 : W[(j + u + 1) & 7]);
            const float2 s1 = __fmul2_rn(B[j], r1);
            const float2 m = (u == 0) ? in[j] : out[j];
            out[j].x = fmax3(m.x, s0.x, s1.x);
            out[j].y = fmax3(m.y, s0.y, s1.y);
        }
        W[u] = n0;
        W[u + 1] = n1;
    }
}

// record, per running sum, whether the block of widths that just ended raised the maximum
__device__ __forceinline__ void note_block(const float2 (&now)[SW_R], const float2 (&old)[SW_R], int w0,
                                           int (&w0x)[SW_R], int (&w0y)[SW_R])
{
#pragma unroll
    for (int j = 0; j < SW_R; ++j) {
        w0x[j] = (now[j].x > old[j].x) ? w0 : w0x[j];
        w0y[j] = (now[j].y > old[j].y) ? w0 : w0y[j];
    }
}

// SNR (f32) and width (u16) of a thread's 8 + 8 samples: 16-byte streaming stores where the row is aligned and whole
template <int SW_THREADS>
__device__ __forceinline__ void store_planes(float *__restrict__ snr, uint16_t *__restrict__ width, int64_t row, int64_t row_stride,
                                             int64_t n_t, int64_t ta, const float2 (&best)[SW_R], const int (&wx)[SW_R], const int (&wy)[SW_R])
{
    const int64_t tb = ta + SW_THREADS * SW_R;
    float *oa = snr + row * row_stride + ta, *ob = snr + row * row_stride + tb;
    const bool v4 = ((reinterpret_cast<uintptr_t>(snr + row * row_stride) & 15) == 0);
    if (v4 && ta + 7 < n_t) {
        __stcs(reinterpret_cast<float4 *>(oa), make_float4(best[0].x, best[1].x, best[2].x, best[3].x));
        __stcs(reinterpret_cast<float4 *>(oa) + 1, make_float4(best[4].x, best[5].x, best[6].x, best[7].x));
    } else {
#pragma unroll
        for (int j = 0; j < SW_R; ++j) if (ta + j < n_t) oa[j] = best[j].x;
    }
    if (v4 && tb + 7 < n_t) {
        __stcs(reinterpret_cast<float4 *>(ob), make_float4(best[0].y, best[1].y, best[2].y, best[3].y));
        __stcs(reinterpret_cast<float4 *>(ob) + 1, make_float4(best[4].y, best[5].y, best[6].y, best[7].y));
    } else {
#pragma unroll
        for (int j = 0; j < SW_R; ++j) if (tb + j < n_t) ob[j] = best[j].y;
    }
    if (width) {
        uint16_t *wa = width + row * row_stride + ta, *wb = width + row * row_stride + tb;
        const bool w8 = ((reinterpret_cast<uintptr_t>(width + row * row_stride) & 15) == 0);
        if (w8 && ta + 7 < n_t)
            __stcs(reinterpret_cast<uint4 *>(wa), make_uint4(wx[0] | (wx[1] << 16), wx[2] | (wx[3] << 16), wx[4] | (wx[5] << 16), wx[6] | (wx[7] << 16)));
        else {
#pragma unroll
            for (int j = 0; j < SW_R; ++j) if (ta + j < n_t) wa[j] = (uint16_t)wx[j];
        }
        if (w8 && tb + 7 < n_t)
            __stcs(reinterpret_cast<uint4 *>(wb), make_uint4(wy[0] | (wy[1] << 16), wy[2] | (wy[3] << 16), wy[4] | (wy[5] << 16), wy[6] | (wy[7] << 16)));
        else {
#pragma unroll
            for (int j = 0; j < SW_R; ++j) if (tb + j < n_t) wb[j] = (uint16_t)wy[j];
        }
    }
}

template <int SW_THREADS>
__global__ void __launch_bounds__(SW_THREADS, 512 / SW_THREADS)
boxcar_snr_sweep(const float *__restrict__ x, int64_t n_t, int64_t row_stride, int tiles_per_row, int64_t total_tiles,
                 const spd_stats_t *__restrict__ st, const float *__restrict__ table, int nmax,
                 float *__restrict__ snr, uint16_t *__restrict__ width)
{
    constexpr int SW_SUB = SW_THREADS * SW_R, SW_TILE = 2 * SW_SUB;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const SweepSmem lay(nmax, SW_THREADS);
    float2 *Z   = reinterpret_cast<float2 *>(smem_raw + lay.z);
    float  *raw = reinterpret_cast<float *>(smem_raw + lay.raw);
    float2 *P2  = reinterpret_cast<float2 *>(smem_raw + lay.p2);      // prefix sums of y: (sub-tile A, sub-tile B), zpad layout
    float2 *scan = reinterpret_cast<float2 *>(smem_raw + lay.scan);   // [2][4] per-warp totals of the tile prefix scan
    float  *rtf = reinterpret_cast<float *>(smem_raw + lay.rtf);      // r_w = 1 / sigma_w

    const int tid = threadIdx.x;
    const int lane = tid & 31, wid = tid >> 5;
    const int nblk = sw_nblk(nmax);
    const int H = sw_halo(nmax);
    const int LRAW = SW_TILE + H;                 // raw floats per tile: x[T0 .. T0 + 2048 + H)
    const int LZ = SW_SUB + H;                    // interleaved positions (a multiple of 8)
    const int nparts = (LZ + SW_SUB - 1) / SW_SUB;
    const double mu = st->mean;
    const float mu_hi = (float)mu, mu_lo = (float)(mu - (double)mu_hi);
    const float2 mu_hi2 = make_float2(-mu_hi, -mu_hi), mu_lo2 = make_float2(-mu_lo, -mu_lo);
    const float NINF = __int_as_float(0xff800000);

    for (int w = tid; w < sw_rt_len(nmax); w += SW_THREADS) rtf[w] = __ldg(table + w);

    int64_t tile = blockIdx.x;
    TilePos pos(blockIdx.x, tiles_per_row);
    __shared__ unsigned long long stage_bar;
    TileStager stg;
    stg.init(&stage_bar, tid);
    if (tile < total_tiles) stg.stage<SW_THREADS, false>(raw, x, n_t, row_stride, pos, LRAW, tid);

    for (; tile < total_tiles; tile += gridDim.x) {
        const int64_t row = pos.row;
        const int64_t T0 = (int64_t)pos.tr * SW_TILE;
        pos = pos.next(gridDim.x, tiles_per_row);                                  // the tile after this one
        stg.wait();
        __syncthreads();                           // raw tile landed; everyone is done with the previous Z / P

        // ---- per-thread state ---------------------------------------------------------------------------------------
        float2 B[SW_R], W[SW_R], bestA[SW_R], bestB[SW_R];
        int w0x[SW_R], w0y[SW_R];
#pragma unroll
        for (int j = 0; j < SW_R; ++j) {
            B[j] = make_float2(0.f, 0.f);
            bestA[j] = make_float2(NINF, NINF);
            w0x[j] = 0; w0y[j] = 0;
        }

        // ---- staging, one pass: every thread takes groups of 8 consecutive positions (part 0: its own 8 samples, whose
        //      y values stay in registers as the first window), forms y = x - mu (two-term fp32 subtract), writes the
        //      interleaved Z and the tile-local inclusive prefix sums P[i + 1] = y[0] + ... + y[i] of both sub-tiles
        //      (only the width search reads P)
        {
            float2 carry = make_float2(0.f, 0.f);
            for (int part = 0; part < nparts; ++part) {
                const int g = part * SW_THREADS + tid;           // group of 8 positions: 8 g .. 8 g + 7
                const bool act = 8 * g < LZ;
                const bool wact = 8 * (g - lane) < LZ;           // warp-uniform: any lane of this warp active (the halo part keeps one warp busy)
                float2 v[SW_R];
                float2 inc = make_float2(0.f, 0.f), off = make_float2(0.f, 0.f);
                float2 *tot = scan + 4 * (part & 1);
                if (wact) {
                    if (act) {
                        const float4 a0 = *reinterpret_cast<const float4 *>(raw + 8 * g), a1 = *reinterpret_cast<const float4 *>(raw + 8 * g + 4);
                        const float4 b0 = *reinterpret_cast<const float4 *>(raw + SW_SUB + 8 * g), b1 = *reinterpret_cast<const float4 *>(raw + SW_SUB + 8 * g + 4);
                        v[0] = make_float2(a0.x, b0.x); v[1] = make_float2(a0.y, b0.y); v[2] = make_float2(a0.z, b0.z); v[3] = make_float2(a0.w, b0.w);
                        v[4] = make_float2(a1.x, b1.x); v[5] = make_float2(a1.y, b1.y); v[6] = make_float2(a1.z, b1.z); v[7] = make_float2(a1.w, b1.w);
#pragma unroll
                        for (int j = 0; j < SW_R; ++j) {
                            v[j] = __fadd2_rn(__fadd2_rn(v[j], mu_hi2), mu_lo2);
                            Z[9 * g + j] = v[j];                 // zpad(8 g + j) = 9 g + j
                        }
                    } else {
#pragma unroll
                        for (int j = 0; j < SW_R; ++j) v[j] = make_float2(0.f, 0.f);
                    }
                    if (part == 0) {
#pragma unroll
                        for (int j = 0; j < SW_R; ++j) W[j] = v[j];
                    }
#pragma unroll
                    for (int j = 1; j < SW_R; ++j) v[j] = __fadd2_rn(v[j], v[j - 1]);
                    inc = v[SW_R - 1];                           // inclusive scan of the thread totals across the warp
#pragma unroll
                    for (int d = 1; d < 32; d <<= 1) {
                        const float ox = __shfl_up_sync(0xffffffffu, inc.x, d), oy = __shfl_up_sync(0xffffffffu, inc.y, d);
                        if (lane >= d) { inc.x += ox; inc.y += oy; }
                    }
                    // exclusive prefix inside the warp (no inc - total: -inf - -inf is NaN)
                    off.x = __shfl_up_sync(0xffffffffu, inc.x, 1); off.y = __shfl_up_sync(0xffffffffu, inc.y, 1);
                    if (lane == 0) off = make_float2(0.f, 0.f);
                }
                if (lane == 31) tot[wid] = inc;
                __syncthreads();                                 // totals visible; this part of raw is consumed, of Z written
                if (part == nparts - 1 && tile + gridDim.x < total_tiles) stg.stage<SW_THREADS, false>(raw, x, n_t, row_stride, pos, LRAW, tid);   // raw is free again
                off = __fadd2_rn(off, carry);
#pragma unroll
                for (int w = 0; w < SW_THREADS / 32; ++w) {
                    const float2 t = tot[w];
                    if (w < wid) off = __fadd2_rn(off, t);
                    carry = __fadd2_rn(carry, t);
                }
                if (act) {
#pragma unroll
                    for (int j = 0; j < SW_R; ++j) P2[zpad(8 * g + j + 1)] = __fadd2_rn(v[j], off);
                }
            }
            if (tid == 0) P2[0] = make_float2(0.f, 0.f);
        }

        // ---- main loop: blocks of 8 widths, the running maximum ping-pongs between bestA and bestB ---------------------
        {
            const float2 *zp = Z + 9 * (tid + 1);                // zpad(8 tid + 8 kb + 8 + u) = 9 (tid + kb + 1) + u
            const float *rp = rtf;
            int kb = 0;
            for (; kb + 2 <= nblk; kb += 2) {
                sweep8(B, W, bestA, bestB, zp, rp);
                note_block(bestB, bestA, 8 * kb, w0x, w0y);
                sweep8(B, W, bestB, bestA, zp + 9, rp + 8);
                note_block(bestA, bestB, 8 * kb + 8, w0x, w0y);
                zp += 18; rp += 16;
            }
            if (kb < nblk) {
                sweep8(B, W, bestA, bestB, zp, rp);
                note_block(bestB, bestA, 8 * kb, w0x, w0y);
#pragma unroll
                for (int j = 0; j < SW_R; ++j) bestA[j] = bestB[j];
            }
        }
        float2 (&best)[SW_R] = bestA;
        __syncthreads();                           // P (written before the main loop) is complete for every warp

        // ---- width search inside the winning block, from the prefix sums: B_w(t) = P[t + w] - P[t] ------------------
        int wx[SW_R], wy[SW_R];
#pragma unroll
        for (int j = 0; j < SW_R; ++j) {
            const float2 p0 = P2[9 * tid + j];                                    // P[t], t = 8 tid + j
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int w0 = h ? w0y[j] : w0x[j];
                const float p0h = h ? p0.y : p0.x;
                const float *pe = reinterpret_cast<const float *>(P2 + 9 * (tid + (w0 >> 3))) + h;   // zpad(8 tid + w0 + c) = 9 (tid + w0/8) + c + (c >> 3)
                const float4 *rq = reinterpret_cast<const float4 *>(rtf + w0);
                const float4 ra = rq[0], rb = rq[1];
                const float r[8] = {ra.x, ra.y, ra.z, ra.w, rb.x, rb.y, rb.z, rb.w};
                float s[8];
#pragma unroll
                for (int g = 0; g < 8; ++g) { const int c = j + g + 1; s[g] = (pe[2 * (c + (c >> 3))] - p0h) * r[g]; }
                // the position inside the block rides in the 3 low mantissa bits (7 - g: ties keep the smallest width);
                // a tagged -inf or NaN (width past the row end / past nmax) is a NaN, which FMNMX drops
#pragma unroll
                for (int g = 0; g < 8; ++g) s[g] = __int_as_float((__float_as_int(s[g]) & ~7) | (7 - g));
                const float m = fmaxf(fmax3(fmax3(s[0], s[1], s[2]), s[3], s[4]), fmax3(s[5], s[6], s[7]));
                const int w = 7 - (__float_as_int(m) & 7);
                if (h) wy[j] = w0 + w + 1; else wx[j] = w0 + w + 1;
            }
        }

        // a NaN reciprocal table (LINEAR mode fed stats of another Nmax) must surface: fmaxf drops NaN operands
        if (rtf[0] != rtf[0]) {
#pragma unroll
            for (int j = 0; j < SW_R; ++j) best[j] = make_float2(rtf[0], rtf[0]);
        }

        store_planes<SW_THREADS>(snr, width, row, row_stride, n_t, T0 + SW_R * tid, best, wx, wy);
    }
    cp_async_commit_wait_all();
}

// ---------------------------------------------------------------------------------------------------------------
// Fused search (spd_search_fused): the same width loop with the threshold of PAPER.md:87-93 applied in
// the kernel.  The planes are never written, so the width is needed at hits only: there is no per-block arg-max
// bookkeeping, no prefix scan and no width search.  A thread that owns a hit replays that one sample's running sums
// in the order of the main loop (same fp32 adds and multiplies, so the values are bit-identical) and takes the first
// width whose SNR equals the maximum: the smallest arg-max (A7).
struct FusedSmem {
    int z, raw, rtf, total;
    __host__ __device__ FusedSmem(int nmax, int nt)
    {
        const int H = sw_halo(nmax), R = sw_rt_len(nmax), SW_SUB = nt * SW_R, SW_TILE = 2 * SW_SUB;
        z = 0;
        raw = z + round_up((zpad(SW_SUB + H) + 1) * 8, 16);
        rtf = raw + round_up((SW_TILE + H) * 4, 16);
        total = rtf + round_up(R * 4, 16);
    }
};

__device__ __noinline__ int replay_width(const float *__restrict__ zh, int pos, const float *__restrict__ rtf, int nmax, float best)
{
    float b = 0.f;
    for (int w = 1; w <= nmax; ++w) {
        b = __fadd_rn(b, zh[2 * zpad(pos + w - 1)]);
        if (__fmul_rn(b, rtf[w - 1]) == best) return w;
    }
    return nmax;                                   // not reached for finite input
}

template <int SW_THREADS>
__global__ void __launch_bounds__(SW_THREADS, 512 / SW_THREADS)
boxcar_search_fused(const float *__restrict__ x, int64_t n_t, int64_t row_stride, int tiles_per_row, int64_t total_tiles,
                    const spd_stats_t *__restrict__ st, const float *__restrict__ table, int nmax,
                    float threshold, spd_candidate_t *__restrict__ cand, unsigned long long capacity,
                    unsigned long long *__restrict__ count)
{
    constexpr int SW_SUB = SW_THREADS * SW_R, SW_TILE = 2 * SW_SUB;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const FusedSmem lay(nmax, SW_THREADS);
    float2 *Z   = reinterpret_cast<float2 *>(smem_raw + lay.z);
    float  *raw = reinterpret_cast<float *>(smem_raw + lay.raw);
    float  *rtf = reinterpret_cast<float *>(smem_raw + lay.rtf);

    const int tid = threadIdx.x;
    const int nblk = sw_nblk(nmax);
    const int H = sw_halo(nmax);
    const int LRAW = SW_TILE + H, LZ = SW_SUB + H;
    const int nparts = (LZ + SW_SUB - 1) / SW_SUB;
    const double mu = st->mean;
    const float mu_hi = (float)mu, mu_lo = (float)(mu - (double)mu_hi);
    const float2 mu_hi2 = make_float2(-mu_hi, -mu_hi), mu_lo2 = make_float2(-mu_lo, -mu_lo);
    const float NINF = __int_as_float(0xff800000);

    for (int w = tid; w < sw_rt_len(nmax); w += SW_THREADS) rtf[w] = __ldg(table + w);

    int64_t tile = blockIdx.x;
    TilePos pos(blockIdx.x, tiles_per_row);
    __shared__ unsigned long long stage_bar;
    TileStager stg;
    stg.init(&stage_bar, tid);
    if (tile < total_tiles) stg.stage<SW_THREADS, false>(raw, x, n_t, row_stride, pos, LRAW, tid);

    for (; tile < total_tiles; tile += gridDim.x) {
        const int64_t row = pos.row;
        const int64_t T0 = (int64_t)pos.tr * SW_TILE;
        pos = pos.next(gridDim.x, tiles_per_row);                                  // the tile after this one
        stg.wait();
        __syncthreads();                           // raw tile landed; everyone is done with the previous Z

        float2 B[SW_R], W[SW_R], best[SW_R];
        for (int part = 0; part < nparts; ++part) {
            const int g = part * SW_THREADS + tid;
            if (8 * g < LZ) {
                const float4 a0 = *reinterpret_cast<const float4 *>(raw + 8 * g), a1 = *reinterpret_cast<const float4 *>(raw + 8 * g + 4);
                const float4 b0 = *reinterpret_cast<const float4 *>(raw + SW_SUB + 8 * g), b1 = *reinterpret_cast<const float4 *>(raw + SW_SUB + 8 * g + 4);
                float2 v[SW_R] = {make_float2(a0.x, b0.x), make_float2(a0.y, b0.y), make_float2(a0.z, b0.z), make_float2(a0.w, b0.w),
                                  make_float2(a1.x, b1.x), make_float2(a1.y, b1.y), make_float2(a1.z, b1.z), make_float2(a1.w, b1.w)};
#pragma unroll
                for (int j = 0; j < SW_R; ++j) {
                    v[j] = __fadd2_rn(__fadd2_rn(v[j], mu_hi2), mu_lo2);
                    Z[9 * g + j] = v[j];
                    if (part == 0) W[j] = v[j];
                }
            }
        }
        __syncthreads();                           // Z complete; raw is free again
        if (tile + gridDim.x < total_tiles) stg.stage<SW_THREADS, false>(raw, x, n_t, row_stride, pos, LRAW, tid);

#pragma unroll
        for (int j = 0; j < SW_R; ++j) { B[j] = make_float2(0.f, 0.f); best[j] = make_float2(NINF, NINF); }
        {
            const float2 *zp = Z + 9 * (tid + 1);
            const float *rp = rtf;
            for (int kb = 0; kb < nblk; ++kb, zp += 9, rp += 8) sweep8(B, W, best, best, zp, rp);
        }

        // ---- threshold; hits replay their own running sums to get the width ------------------------------------------
        const int64_t ta = T0 + SW_R * tid, tb = ta + SW_SUB;
        bool any = false;
#pragma unroll
        for (int j = 0; j < SW_R; ++j) any |= (best[j].x >= threshold && ta + j < n_t) || (best[j].y >= threshold && tb + j < n_t);
        if (__any_sync(0xffffffffu, any)) {
            const float *zf = reinterpret_cast<const float *>(Z);
#pragma unroll
            for (int j = 0; j < SW_R; ++j) {
                const bool ha = best[j].x >= threshold && ta + j < n_t;
                const bool hb = best[j].y >= threshold && tb + j < n_t;
                int wa = 1, wb = 1;
                if (ha) wa = replay_width(zf, SW_R * tid + j, rtf, nmax, best[j].x);
                if (hb) wb = replay_width(zf + 1, SW_R * tid + j, rtf, nmax, best[j].y);
                __syncwarp();
                append_candidate(ha, (uint32_t)row, (uint32_t)(ta + j), best[j].x, (uint32_t)wa, cand, capacity, count);
                append_candidate(hb, (uint32_t)row, (uint32_t)(tb + j), best[j].y, (uint32_t)wb, cand, capacity, count);
            }
        }
    }
    cp_async_commit_wait_all();
}

// ---------------------------------------------------------------------------------------------------------------
// Narrow searches (nmax <= SW_NARROW_NMAX; the tag has room for 32 widths): the fixed per-sample cost of the general kernel (prefix scan + width search, about 100
// clocks per 32 samples) is larger than the width loop itself, so here the arg-max rides along with the maximum:
// beside the exact running maximum a second one is kept over TAGGED values, (bits(s) & ~31) | (32 - w).  A larger
// tag is a smaller width, so exact ties keep the smallest width (A7); values closer than 32 ulp (4e-6 relative, far
// inside the 1e-3 tie tolerance of DESIGN.md section 5) may resolve either way.  The SNR written is the exact maximum.
// A tagged -inf (a window past the row end) is a NaN, which FMNMX drops.  No scan, no width search, no bookkeeping.
template <int KB>
__device__ __forceinline__ void sweep8_tagged(float2 (&B)[SW_R], float2 (&W)[SW_R], float2 (&best)[SW_R], float2 (&tbest)[SW_R],
                                              const float2 *__restrict__ zp, const float *__restrict__ rp)
{
#pragma unroll
    for (int u = 0; u < 8; u += 2) {
        const float2 rr = *reinterpret_cast<const float2 *>(rp + u);
        const float2 r0 = make_float2(rr.x, rr.x), r1 = make_float2(rr.y, rr.y);
        const float2 n0 = zp[u], n1 = zp[u + 1];
        constexpr int MASK = ~31;
        const int c0 = 32 - (8 * KB + u + 1), c1 = c0 - 1;              // 32 - w for the two widths of this step
#pragma unroll
        for (int j = 0; j < SW_R; ++j) {
            B[j] = __fadd2_rn(B[j], W[(j + u) & 7]);
            const float2 s0 = __fmul2_rn(B[j], r0);
            B[j] = __fadd2_rn(B[j], (j == SW_R - 1) ? n0 : W[(j + u + 1) & 7]);
            const float2 s1 = __fmul2_rn(B[j], r1);
            best[j].x = fmax3(best[j].x, s0.x, s1.x);
            best[j].y = fmax3(best[j].y, s0.y, s1.y);
            tbest[j].x = fmax3(tbest[j].x, __int_as_float((__float_as_int(s0.x) & MASK) | c0), __int_as_float((__float_as_int(s1.x) & MASK) | c1));
            tbest[j].y = fmax3(tbest[j].y, __int_as_float((__float_as_int(s0.y) & MASK) | c0), __int_as_float((__float_as_int(s1.y) & MASK) | c1));
        }
        W[u] = n0;
        W[u + 1] = n1;
    }
}

template <int SW_THREADS>
__global__ void __launch_bounds__(SW_THREADS, 640 / SW_THREADS)
boxcar_snr_sweep_narrow(const float *__restrict__ x, int64_t n_t, int64_t row_stride, int tiles_per_row, int64_t total_tiles,
                        const spd_stats_t *__restrict__ st, const float *__restrict__ table, int nmax,
                        float *__restrict__ snr, uint16_t *__restrict__ width)
{
    constexpr int SW_SUB = SW_THREADS * SW_R, SW_TILE = 2 * SW_SUB;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const FusedSmem lay(nmax, SW_THREADS);
    float2 *Z   = reinterpret_cast<float2 *>(smem_raw + lay.z);
    float  *raw = reinterpret_cast<float *>(smem_raw + lay.raw);
    float  *rtf = reinterpret_cast<float *>(smem_raw + lay.rtf);

    const int tid = threadIdx.x;
    const int nblk = sw_nblk(nmax);
    const int H = sw_halo(nmax);
    const int LRAW = SW_TILE + H, LZ = SW_SUB + H;
    const int nparts = (LZ + SW_SUB - 1) / SW_SUB;
    const double mu = st->mean;
    const float mu_hi = (float)mu, mu_lo = (float)(mu - (double)mu_hi);
    const float2 mu_hi2 = make_float2(-mu_hi, -mu_hi), mu_lo2 = make_float2(-mu_lo, -mu_lo);
    const float NINF = __int_as_float(0xff800000);

    for (int w = tid; w < sw_rt_len(nmax); w += SW_THREADS) rtf[w] = __ldg(table + w);

    int64_t tile = blockIdx.x;
    TilePos pos(blockIdx.x, tiles_per_row);
    __shared__ unsigned long long stage_bar;
    TileStager stg;
    stg.init(&stage_bar, tid);
    if (tile < total_tiles) stg.stage<SW_THREADS, true>(raw, x, n_t, row_stride, pos, LRAW, tid);

    for (; tile < total_tiles; tile += gridDim.x) {
        const int64_t row = pos.row;
        const int64_t T0 = (int64_t)pos.tr * SW_TILE;
        pos = pos.next(gridDim.x, tiles_per_row);                                  // the tile after this one
        stg.wait();
        __syncthreads();                           // raw tile landed; everyone is done with the previous Z

        float2 B[SW_R], W[SW_R], best[SW_R], tbest[SW_R];
        for (int part = 0; part < nparts; ++part) {
            const int g = part * SW_THREADS + tid;
            if (8 * g < LZ) {
                const float4 a0 = *reinterpret_cast<const float4 *>(raw + 8 * g), a1 = *reinterpret_cast<const float4 *>(raw + 8 * g + 4);
                const float4 b0 = *reinterpret_cast<const float4 *>(raw + SW_SUB + 8 * g), b1 = *reinterpret_cast<const float4 *>(raw + SW_SUB + 8 * g + 4);
                float2 v[SW_R] = {make_float2(a0.x, b0.x), make_float2(a0.y, b0.y), make_float2(a0.z, b0.z), make_float2(a0.w, b0.w),
                                  make_float2(a1.x, b1.x), make_float2(a1.y, b1.y), make_float2(a1.z, b1.z), make_float2(a1.w, b1.w)};
#pragma unroll
                for (int j = 0; j < SW_R; ++j) {
                    v[j] = __fadd2_rn(__fadd2_rn(v[j], mu_hi2), mu_lo2);
                    Z[9 * g + j] = v[j];
                    if (part == 0) W[j] = v[j];
                }
            }
        }
        __syncthreads();                           // Z complete; raw is free again
        if (tile + gridDim.x < total_tiles) stg.stage<SW_THREADS, true>(raw, x, n_t, row_stride, pos, LRAW, tid);

#pragma unroll
        for (int j = 0; j < SW_R; ++j) { B[j] = make_float2(0.f, 0.f); best[j] = make_float2(NINF, NINF); tbest[j] = make_float2(NINF, NINF); }
        const float2 *zp = Z + 9 * (tid + 1);
        sweep8_tagged<0>(B, W, best, tbest, zp, rtf);
        if (nblk > 1) sweep8_tagged<1>(B, W, best, tbest, zp + 9, rtf + 8);
        if (nblk > 2) sweep8_tagged<2>(B, W, best, tbest, zp + 18, rtf + 16);
        if (nblk > 3) sweep8_tagged<3>(B, W, best, tbest, zp + 27, rtf + 24);

        int wx[SW_R], wy[SW_R];
#pragma unroll
        for (int j = 0; j < SW_R; ++j) { wx[j] = 32 - (__float_as_int(tbest[j].x) & 31); wy[j] = 32 - (__float_as_int(tbest[j].y) & 31); }
        if (rtf[0] != rtf[0]) {                     // NaN table (LINEAR mode fed stats of another Nmax) must surface
#pragma unroll
            for (int j = 0; j < SW_R; ++j) { best[j] = make_float2(rtf[0], rtf[0]); wx[j] = 1; wy[j] = 1; }
        }
        store_planes<SW_THREADS>(snr, width, row, row_stride, n_t, T0 + SW_R * tid, best, wx, wy);
    }
    cp_async_commit_wait_all();
}

template <typename K>
static cudaError_t persistent_grid(K kernel, int threads, int smem, int64_t tiles, unsigned *grid)
{
    cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return e;
    int dev = 0, sms = 0, per_sm = 0;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
    if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
    if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, threads, smem)) != cudaSuccess) return e;
    if (per_sm < 1) return cudaErrorInvalidConfiguration;
    const int64_t wave = (int64_t)sms * per_sm;                 // persistent: one resident wave walks all tiles
    *grid = (unsigned)(tiles < wave ? tiles : wave);
    return cudaSuccess;
}

template <int NT>
static cudaError_t launch_sweep_nt(const float *x, int64_t n_dm, int64_t n_t, int64_t row_stride, const spd_stats_t *d_stats,
                                   const float *d_table, int nmax, float *snr, uint16_t *width,
                                   bool fused, float threshold, spd_candidate_t *out, unsigned long long capacity,
                                   unsigned long long *d_count, cudaStream_t s)
{
    constexpr int TILE = 2 * NT * SW_R;
    const int tpr = (int)((n_t + TILE - 1) / TILE);
    const int64_t tiles = n_dm * (int64_t)tpr;
    unsigned grid = 0;
    cudaError_t e;
    if (fused) {
        const FusedSmem lay(nmax, NT);
        if ((e = persistent_grid(boxcar_search_fused<NT>, NT, lay.total, tiles, &grid)) != cudaSuccess) return e;
        boxcar_search_fused<NT><<<grid, NT, lay.total, s>>>(x, n_t, row_stride, tpr, tiles, d_stats, d_table, nmax,
                                                            threshold, out, capacity, d_count);
    } else if (nmax <= SW_NARROW_NMAX) {
        const FusedSmem lay(nmax, NT);
        if ((e = persistent_grid(boxcar_snr_sweep_narrow<NT>, NT, lay.total, tiles, &grid)) != cudaSuccess) return e;
        boxcar_snr_sweep_narrow<NT><<<grid, NT, lay.total, s>>>(x, n_t, row_stride, tpr, tiles, d_stats, d_table, nmax, snr, width);
    } else {
        const SweepSmem lay(nmax, NT);
        if ((e = persistent_grid(boxcar_snr_sweep<NT>, NT, lay.total, tiles, &grid)) != cudaSuccess) return e;
        boxcar_snr_sweep<NT><<<grid, NT, lay.total, s>>>(x, n_t, row_stride, tpr, tiles, d_stats, d_table, nmax, snr, width);
    }
    return cudaGetLastError();
}

cudaError_t launch_sweep(const float *x, int64_t n_dm, int64_t n_t, int64_t row_stride, const spd_stats_t *d_stats,
                         const float *d_table, int nmax, float *snr, uint16_t *width,
                         bool fused, float threshold, spd_candidate_t *out, unsigned long long capacity,
                         unsigned long long *d_count, cudaStream_t s)
{
    if (nmax <= SW_SMALL_CTA_NMAX)
        return launch_sweep_nt<64>(x, n_dm, n_t, row_stride, d_stats, d_table, nmax, snr, width, fused, threshold, out, capacity, d_count, s);
    return launch_sweep_nt<128>(x, n_dm, n_t, row_stride, d_stats, d_table, nmax, snr, width, fused, threshold, out, capacity, d_count, s);
}

}  // namespace spd
