// sweep.cu -- steps 2-4a: boxcars of every width, SNR, max / arg-max over width, one kernel
// (section 2.3, Algorithm 1; readings A5-A9 of DESIGN.md).
//
//   B_N(t) = sum_{k<N} x[t+k];  SNR_N(t) = (B_N(t) - N mu) / sigma_N;  snr[t] = max_N, width[t] = smallest arg-max.
//
// Four kernels share one width loop (sweep8 / sweep8_tagged): boxcar_snr_sweep (planes, any nmax), boxcar_snr_sweep_narrow
// (planes, nmax <= 32; also one level of the decimated search), boxcar_search_fused (threshold in the kernel, no planes) and
// boxcar_search_fused_level (the same for one level of the decimated search).
//
// What bounds the loop (measured with a microbenchmark, profiles/r02_fp32_issue_rates.md): one warp instruction per
// sub-partition per clock, a packed FADD2 / FMUL2 counts as two (it passes the 32-lane FMA pipe twice), an ALU-pipe
// instruction (FMNMX3, LOP3, FSETP, SEL) occupies its 16-lane pipe for two clocks.  One (sample, width) pair needs an add,
// a multiply and half a 3-input maximum = 2.5 issue slots; everything else in this file exists to add as little as
// possible to that.
//
// Design (sm_100a; this is NOT the paper's one-thread-X-samples loop):
//  * Persistent CTAs (one wave, grid = SMs x resident CTAs) walk the tiles; the raw samples of the NEXT tile are
//    prefetched with cp.async (LDGSTS, 16 B) or one 1-D TMA bulk copy into shared memory while the current tile is swept.
//  * y = x - mu is formed once per sample when the raw tile is converted into the working layout (two-term fp32
//    subtract, mu = mu_hi + mu_lo), so the inner loop is B += y; s = B * r_N.
//  * Where r_N comes from (template parameter RC):
//      RC = true  (eq. 4 and nmax a multiple of 8): y is also divided by sigma once per sample, and r_N = 1/sqrt(N)
//                 is read from a compile-time table in the CONSTANT bank, so it reaches FMUL2 as a uniform-register
//                 operand: one register-file read less per multiply (measured 2.8 -> 2.5 clocks per pair).
//      RC = false (eq. 5 modes, any nmax): r_N = 1/sigma_N from the table sigma_table_kernel wrote, staged in shared
//                 memory and fed as a scalar-broadcast register operand.
//  * One tile = 16 NT consecutive samples of one row, as two sub-tiles A = [T0, T0 + 8 NT), B = [T0 + 8 NT, T0 + 16 NT).
//    The working layout INTERLEAVES them, float2 Z[i] = (yA[i], yB[i]), so that one packed FADD2 / FMUL2 advances one
//    running sum of each sub-tile.
//  * Each thread owns 8 consecutive samples of each sub-tile and keeps a sliding window of 8 float2 in registers
//    (the width loop is unrolled by 8, so the rotation is register renaming): one LDS.128 per two width steps.
//  * y is formed on the register pairs the 16-byte loads of the raw tile deliver (two consecutive samples of one
//    sub-tile), the last step scalar, so the interleaved pairs need no register moves (Norm::apply_pair).
//  * Samples past the row end are staged as -inf: a running sum that has touched one is -inf for every wider
//    width, so "only widths that fit" (reading A9) needs no masking in the loop.  In the RC = false kernels widths
//    nmax < w <= 8 ceil(nmax/8) get a NaN reciprocal: FMNMX drops NaN operands, so they can never win.
//  * arg-max of the general kernel is deferred: the running maximum is advanced with 3-input FMNMX only,
//    ping-ponging between two register sets so that the value before and after each block of 8 widths are both
//    live; one compare + one select per block then record the block that last raised it.  After the loop that block
//    alone is evaluated again from tile-local prefix sums E kept in shared memory (B_w(t) = E[t+w] - E[t], no
//    dependency chain); the position inside the block rides in the 3 low mantissa bits of the 8 values (a larger tag
//    is a smaller width), so one maximum gives the width.  Blocks ascend with a strict '>', so exact ties keep the
//    smallest width (A7) for non-negative maxima.  The SNR written is the running-sum value of the main loop; the
//    re-evaluation only picks the width and differs from the running sums by fp32 rounding and the 3 tag bits (~1e-6
//    relative), i.e. only inside near-ties far below the 1e-3 tie tolerance.
//
// Roofline: 10 B/sample of HBM traffic (4 read + 4 snr + 2 width) against 2 Nmax FMA-pipe lane-ops per sample
// (SURVEY.md 8(d)); FP32-issue-bound for Nmax > ~24.
#include "spd_common.cuh"

#include <mutex>

namespace spd {

constexpr int SW_R       = 8;                        // samples per thread per sub-tile
// CTA width NT (a template parameter of the kernels): sub-tile = 8 NT samples, tile = 16 NT samples of one row.
// 64 threads (tile 1024) for nmax <= SW_SMALL_CTA_NMAX: fewer warps wait on each block barrier; 128 threads (tile 2048)
// above, where the halo (nmax + 8 positions staged and scanned per tile) would weigh too much on a small tile.
// The general plane kernel runs ONE-warp CTAs (tile 512) up to SW_WARP_CTA_NMAX: its three block barriers per tile then
// cost nothing (measured on the config-3 shape: Nmax 64 12.87 -> 12.54 ms, Nmax 128 20.39 -> 20.09 ms; Nmax 256 is slower,
// and the fused and narrow kernels, which have a single barrier per tile, do not move).
constexpr int SW_SMALL_CTA_NMAX = 256;
constexpr int SW_WARP_CTA_NMAX = 128;
constexpr int SW_NARROW_NMAX = 32;                   // nmax up to here takes the tagged-maximum kernel (5 tag bits)
constexpr int SW_NMAX_TAB = 4096 + 16;               // entries of the constant 1/sqrt(w) table (API limit of nmax + padding)

__host__ __device__ inline int zpad(int i) { return i + ((i >> 3) << 1); }   // two pad float2 per 8: lane stride 80 B, conflict-free 16-byte accesses
__host__ __device__ inline int sw_nblk(int nmax) { return (nmax + 7) >> 3; }  // blocks of 8 widths
__host__ __device__ inline int sw_halo(int nmax) { return 8 * sw_nblk(nmax) + 8; }   // positions staged past a sub-tile
__host__ __device__ inline int sw_rt_len(int nmax) { return 8 * sw_nblk(nmax) + 8; } // reciprocal-table entries

size_t sweep_table_bytes(int nmax) { return (size_t)sw_rt_len(nmax) * sizeof(float); }

// ---- 1/sqrt(w), w = 1.., as a compile-time table in the constant bank (eq. 4: sigma_N = sqrt(N) sigma) ----
struct IsqrtTable { float v[SW_NMAX_TAB]; };
constexpr double sw_csqrt(double x) { double g = x > 1.0 ? x : 1.0; for (int i = 0; i < 64; ++i) g = 0.5 * (g + x / g); return g; }
constexpr IsqrtTable sw_make_isqrt() { IsqrtTable t{}; for (int i = 0; i < SW_NMAX_TAB; ++i) t.v[i] = (float)(1.0 / sw_csqrt((double)(i + 1))); return t; }
__constant__ IsqrtTable c_isqrt = sw_make_isqrt();

struct SweepSmem {           // byte offsets into dynamic shared memory (all 16-byte aligned)
    int z, raw, ea, eb, scan, rtf, total;
    __host__ __device__ SweepSmem(int nmax, int nt)
    {
        const int H = sw_halo(nmax), R = sw_rt_len(nmax), SW_SUB = nt * SW_R, SW_TILE = 2 * SW_SUB;
        const int groups = (SW_SUB + H) / 8 + 1;                         // groups of 8 prefix sums, 12 floats apart (48 B: conflict-free LDS.128)
        z = 0;                                                           // float2 Z[zpad(SUB + H)]
        raw = z + round_up((zpad(SW_SUB + H) + 1) * 8, 16);              // float raw[TILE + H]
        ea = raw + round_up((SW_TILE + H) * 4, 16);                      // float EA[groups][12]: exclusive prefix sums of sub-tile A
        eb = ea + groups * 48;                                           // float EB[groups][12]
        scan = eb + groups * 48;                                         // float2 [2][4]: per-warp totals of the scan (double-buffered by part)
        rtf = scan + 64;                                                 // float r_w
        total = rtf + round_up(R * 4, 16);
    }
};

__device__ __forceinline__ float fmax3(float a, float b, float c) { return fmaxf(fmaxf(a, b), c); }

// (a & mask) | tag in ONE LOP3 (mask must live in a register: with two immediates the compiler emits two instructions)
__device__ __forceinline__ float tag_bits(float s, int mask, int tag)
{
    int d;
    asm("lop3.b32 %0, %1, %2, %3, 0xEA;" : "=r"(d) : "r"(__float_as_int(s)), "r"(mask), "r"(tag));
    return __int_as_float(d);
}
__device__ __forceinline__ int opaque_reg(int v) { asm volatile("mov.b32 %0, %0;" : "+r"(v)); return v; }

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
// Decimated levels (spd_boxcar_snr_decimated): entry w' - 1 holds 1/sigma_N of the EFFECTIVE width N = w' * wscale, with
// sigma_N of the exhaustive search of nmax_total = the widest effective width (st holds the statistics of the ORIGINAL x).
__global__ void sigma_table_kernel(const spd_stats_t *__restrict__ st, int nmax, int mode, float *__restrict__ table,
                                   int wscale, int nmax_total)
{
    st += blockIdx.y;                               // per-row statistics: one table per row (grid.y = rows, else 1)
    table += (size_t)blockIdx.y * sw_rt_len(nmax);
    const double sigma = st->sigma, snm = st->sigma_nmax;
    const bool bad = (mode != SPD_SIGMA_SQRT) && (st->nmax_of_sigma != nmax_total);
    for (int w = 1 + blockIdx.x * blockDim.x + threadIdx.x; w <= sw_rt_len(nmax); w += gridDim.x * blockDim.x) {
        float r = __int_as_float(0x7fc00000);      // widths past nmax (padding of the last block of 8) never win
        if (w <= nmax) {
            const double N = (double)w * (double)wscale;
            double s = sqrt(N) * sigma;
            if (mode == SPD_SIGMA_LINEAR && nmax_total > 1) s += (N - 1.0) * snm / (double)(nmax_total - 1);
            if (mode == SPD_SIGMA_LINEAR_ANCHORED && nmax_total > 1)
                s += (N - 1.0) * (snm - sqrt((double)nmax_total) * sigma) / (double)(nmax_total - 1);
            r = bad ? __int_as_float(0x7fc00000) : (float)(1.0 / s);
        }
        table[w - 1] = r;
    }
}

cudaError_t launch_sigma_table(const spd_stats_t *d_stats, int nmax, int mode, float *d_table, cudaStream_t s, int wscale, int nmax_total,
                               int64_t rows)
{
    int n = sw_rt_len(nmax);
    for (int64_t r0 = 0; r0 < rows; r0 += 65535) {               // grid.y limit
        const unsigned ny = (unsigned)(rows - r0 < 65535 ? rows - r0 : 65535);
        sigma_table_kernel<<<dim3((n + 255) / 256, ny), 256, 0, s>>>(d_stats + r0, nmax, mode, d_table + (size_t)r0 * n, wscale,
                                                                      nmax_total > 0 ? nmax_total : nmax);
    }
    return cudaGetLastError();
}

// ---- decimation in time (reading A20): x_l[i] = x_{l-1}[2i] + x_{l-1}[2i+1]; the statistics of a level are those
// of x scaled to sums of D = 2^l samples: mean_l = D mu, sigma_l = sqrt(D) sigma (eq. 3), so that eq. 4 of the decimated
// series at width w' IS eq. 4 of x at the effective width w' D.  Nothing is re-measured.
// The level kernels carry the series with the mean already taken out (level 0 subtracts mu from every sample before it
// forms the pair sums, Norm::apply_pair_sum), so above level 0 the mean handed to the kernel is 0, not D mu.
__global__ void level_stats_kernel(const spd_stats_t *__restrict__ st, int D, spd_stats_t *__restrict__ out)
{
    spd_stats_t s = *st;
    s.mean = D == 1 ? st->mean : 0.0;
    s.sigma = st->sigma * sqrt((double)D);
    *out = s;
}

cudaError_t launch_level_stats(const spd_stats_t *st, int D, spd_stats_t *out, cudaStream_t s)
{
    level_stats_kernel<<<1, 1, 0, s>>>(st, D, out);
    return cudaGetLastError();
}

bool sweep_uses_constant_table(int nmax, int mode) { return mode == SPD_SIGMA_SQRT && (nmax & 7) == 0; }

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
// otherwise every thread issues 16-byte cp.async.  Tiles that touch the row end, and rows that are not 16-byte aligned,
// are staged by all threads (cp.async 16 B where possible, scalar loads otherwise; samples past the row end become -inf).
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

// What every sweep kernel needs from the statistics: y = ((x - mu_hi) - mu_lo) [* 1/sigma when RC]
struct Norm {
    float2 mu_hi2, mu_lo2, rs2;
    __device__ __forceinline__ Norm(const spd_stats_t *st) { load(st); }
    __device__ __forceinline__ void load(const spd_stats_t *st)
    {
        const double mu = st->mean;
        const float mu_hi = (float)mu, mu_lo = (float)(mu - (double)mu_hi), rs = (float)(1.0 / st->sigma);
        mu_hi2 = make_float2(-mu_hi, -mu_hi); mu_lo2 = make_float2(-mu_lo, -mu_lo); rs2 = make_float2(rs, rs);
    }
    template <bool RC>
    __device__ __forceinline__ float2 apply(float2 v) const
    {
        v = __fadd2_rn(__fadd2_rn(v, mu_hi2), mu_lo2);
        return RC ? __fmul2_rn(v, rs2) : v;
    }
    // the same arithmetic for two CONSECUTIVE raw samples (p, q) of one sub-tile, as they sit in the registers of a 16-byte
    // load: the packed steps run on that native pair and the last step is scalar, so the results can be written straight
    // into the interleaved (sub-tile A, sub-tile B) pairs without register moves (same issue slots: a packed op takes two)
    template <bool RC>
    __device__ __forceinline__ void apply_pair(float p, float q, float &op, float &oq) const
    {
        float2 v = __fadd2_rn(make_float2(p, q), mu_hi2);
        if (RC) {
            v = __fadd2_rn(v, mu_lo2);
            op = __fmul_rn(v.x, rs2.x); oq = __fmul_rn(v.y, rs2.x);
        } else {
            op = __fadd_rn(v.x, mu_lo2.x); oq = __fadd_rn(v.y, mu_lo2.x);
        }
    }
    // apply_pair, and sum = y_p + y_q of the mean-subtracted samples BEFORE the 1/sigma scaling: one sample of the next
    // decimated level.  Summing y instead of the raw x keeps the level series at the size of the noise, not of D mu
    // (a baseline of 1e3 sigma would otherwise cost ulp(D mu) per level in every SNR above level 0).
    template <bool RC>
    __device__ __forceinline__ void apply_pair_sum(float p, float q, float &op, float &oq, float &sum) const
    {
        float2 v = __fadd2_rn(make_float2(p, q), mu_hi2);
        if (RC) {
            v = __fadd2_rn(v, mu_lo2);
            sum = __fadd_rn(v.x, v.y);
            op = __fmul_rn(v.x, rs2.x); oq = __fmul_rn(v.y, rs2.x);
        } else {
            op = __fadd_rn(v.x, mu_lo2.x); oq = __fadd_rn(v.y, mu_lo2.x);
            sum = __fadd_rn(op, oq);
        }
    }
};

// 8 groups of one raw tile -> 8 interleaved values (sub-tile A, sub-tile B) of group g
template <int SW_SUB>
__device__ __forceinline__ void load_group(const float *raw, int g, float2 (&v)[SW_R])
{
    const float4 a0 = *reinterpret_cast<const float4 *>(raw + 8 * g), a1 = *reinterpret_cast<const float4 *>(raw + 8 * g + 4);
    const float4 b0 = *reinterpret_cast<const float4 *>(raw + SW_SUB + 8 * g), b1 = *reinterpret_cast<const float4 *>(raw + SW_SUB + 8 * g + 4);
    v[0] = make_float2(a0.x, b0.x); v[1] = make_float2(a0.y, b0.y); v[2] = make_float2(a0.z, b0.z); v[3] = make_float2(a0.w, b0.w);
    v[4] = make_float2(a1.x, b1.x); v[5] = make_float2(a1.y, b1.y); v[6] = make_float2(a1.z, b1.z); v[7] = make_float2(a1.w, b1.w);
}

// the same with y = x - mu (and / sigma) formed on the way (Norm::apply_pair)
template <int SW_SUB, bool RC, bool PAIRSUMS = false>
__device__ __forceinline__ void load_norm_group(const float *raw, int g, const Norm &norm, float2 (&v)[SW_R], float4 *sa = nullptr, float4 *sb = nullptr)
{
    const float4 a0 = *reinterpret_cast<const float4 *>(raw + 8 * g), a1 = *reinterpret_cast<const float4 *>(raw + 8 * g + 4);
    const float4 b0 = *reinterpret_cast<const float4 *>(raw + SW_SUB + 8 * g), b1 = *reinterpret_cast<const float4 *>(raw + SW_SUB + 8 * g + 4);
    if (PAIRSUMS) {                                   // x'[i] = y[2i] + y[2i+1], y = x - mu (decimation in time; the level's mean is then 0)
        norm.apply_pair_sum<RC>(a0.x, a0.y, v[0].x, v[1].x, sa->x); norm.apply_pair_sum<RC>(a0.z, a0.w, v[2].x, v[3].x, sa->y);
        norm.apply_pair_sum<RC>(a1.x, a1.y, v[4].x, v[5].x, sa->z); norm.apply_pair_sum<RC>(a1.z, a1.w, v[6].x, v[7].x, sa->w);
        norm.apply_pair_sum<RC>(b0.x, b0.y, v[0].y, v[1].y, sb->x); norm.apply_pair_sum<RC>(b0.z, b0.w, v[2].y, v[3].y, sb->y);
        norm.apply_pair_sum<RC>(b1.x, b1.y, v[4].y, v[5].y, sb->z); norm.apply_pair_sum<RC>(b1.z, b1.w, v[6].y, v[7].y, sb->w);
        return;
    }
    norm.apply_pair<RC>(a0.x, a0.y, v[0].x, v[1].x); norm.apply_pair<RC>(a0.z, a0.w, v[2].x, v[3].x);
    norm.apply_pair<RC>(a1.x, a1.y, v[4].x, v[5].x); norm.apply_pair<RC>(a1.z, a1.w, v[6].x, v[7].x);
    norm.apply_pair<RC>(b0.x, b0.y, v[0].y, v[1].y); norm.apply_pair<RC>(b0.z, b0.w, v[2].y, v[3].y);
    norm.apply_pair<RC>(b1.x, b1.y, v[4].y, v[5].y); norm.apply_pair<RC>(b1.z, b1.w, v[6].y, v[7].y);
}

// group g of the working layout: Z[zpad(8 g + j)] = v[j], four 16-byte stores (zpad(8 g) = 10 g)
__device__ __forceinline__ void store_group(float2 *Z, int g, const float2 (&v)[SW_R])
{
    float4 *d = reinterpret_cast<float4 *>(Z + 10 * g);
#pragma unroll
    for (int k = 0; k < 4; ++k) d[k] = make_float4(v[2 * k].x, v[2 * k].y, v[2 * k + 1].x, v[2 * k + 1].y);
}

// One block of 8 width steps: advance the 8 packed running sums, scale, fold into the running maxima.
// out[j] = max(in[j], the 8 SNRs of this block); `in` stays intact so that the caller can tell whether the block
// raised the maximum.  On entry W[v] = Z[8 tid + a0 + v] (a0 = width offset of the first step); on exit the window
// has moved by 8.  zp -> Z[8 (tid + kb + 1)] (the next 8 window elements).  r_w of the block: RC -> c_isqrt.v[w0 + u]
// (w0 = 8 kb, warp-uniform: a uniform-register operand of FMUL2); otherwise rp[u] from shared memory (a scalar-broadcast
// register operand: FMUL2 broadcasts one register to both halves, one register read less than a (r_w, r_w) pair).
template <bool RC>
__device__ __forceinline__ void sweep8(float2 (&B)[SW_R], float2 (&W)[SW_R], const float2 (&in)[SW_R], float2 (&out)[SW_R],
                                       const float2 *__restrict__ zp, const float *__restrict__ rp, int w0)
{
#pragma unroll
    for (int u = 0; u < 8; u += 2) {
        float2 rr;
        if (RC) rr = make_float2(c_isqrt.v[w0 + u], c_isqrt.v[w0 + u + 1]);
        else rr = *reinterpret_cast<const float2 *>(rp + u);
        const float2 r0 = make_float2(rr.x, rr.x), r1 = make_float2(rr.y, rr.y);
        const float4 nq = *reinterpret_cast<const float4 *>(zp + u);     // two window elements per 16-byte load
        const float2 n0 = make_float2(nq.x, nq.y), n1 = make_float2(nq.z, nq.w);
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

// record, per running sum, whether the block of widths that just ended raised the maximum (kb = index of the block)
__device__ __forceinline__ void note_block(const float2 (&now)[SW_R], const float2 (&old)[SW_R], int kb,
                                           int (&kx)[SW_R], int (&ky)[SW_R])
{
#pragma unroll
    for (int j = 0; j < SW_R; ++j) {
        kx[j] = (now[j].x > old[j].x) ? kb : kx[j];
        ky[j] = (now[j].y > old[j].y) ? kb : ky[j];
    }
}

// SNR (f32) and width (u16) of a thread's 8 + 8 samples: 16-byte streaming stores where the row is aligned and whole
template <int SW_THREADS>
__device__ __forceinline__ void store_planes(float *__restrict__ snr, uint16_t *__restrict__ width, int64_t row, int64_t row_stride /* of the planes */,
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

// Width inside the winning block of ONE sample (position J of the thread's 8, J a compile-time constant), from the
// exclusive prefix sums E of its sub-tile: B_w(t) = E[t + w] - E[t].  E is kept in groups of 8 (12 floats apart), group
// G = tid + kb holds E[8 tid + 8 kb ..+7], so the 8 candidates E[t + 8 kb + 1 .. + 8] are elements J+1..7 of group G
// and 0..J of group G + 1: at most four 16-byte loads, no address arithmetic per candidate.  The position inside the
// block rides in the 3 low mantissa bits (7 - g: exact ties keep the smallest width); a tagged -inf or NaN (width
// past the row end / past nmax) is a NaN, which FMNMX drops.
template <int J>
__device__ __forceinline__ int width_in_block(const float *__restrict__ E, const float *__restrict__ rtf, int tid, int kb, float p0, int mask)
{
    const float4 *eg = reinterpret_cast<const float4 *>(E + (tid + kb) * 12);       // group G; G + 1 is 3 float4 further
    float e[16];
    if (J + 1 < 4) { const float4 q = eg[0]; e[0] = q.x; e[1] = q.y; e[2] = q.z; e[3] = q.w; }
    if (J + 1 < 8) { const float4 q = eg[1]; e[4] = q.x; e[5] = q.y; e[6] = q.z; e[7] = q.w; }
    { const float4 q = eg[3]; e[8] = q.x; e[9] = q.y; e[10] = q.z; e[11] = q.w; }
    if (J >= 4) { const float4 q = eg[4]; e[12] = q.x; e[13] = q.y; e[14] = q.z; e[15] = q.w; }
    const float4 *rq = reinterpret_cast<const float4 *>(rtf + 8 * kb);
    const float4 ra = rq[0], rb = rq[1];
    const float r[8] = {ra.x, ra.y, ra.z, ra.w, rb.x, rb.y, rb.z, rb.w};
    float s[8];
#pragma unroll
    for (int g = 0; g < 8; ++g) s[g] = tag_bits((e[J + 1 + g] - p0) * r[g], mask, 7 - g);
    const float m = fmaxf(fmax3(fmax3(s[0], s[1], s[2]), s[3], s[4]), fmax3(s[5], s[6], s[7]));
    return 8 * kb + 8 - (__float_as_int(m) & 7);
}

template <int SW_THREADS, bool RC>
__global__ void __launch_bounds__(SW_THREADS, 512 / SW_THREADS)
boxcar_snr_sweep(const float *__restrict__ x, int64_t n_t, int64_t row_stride, int tiles_per_row, int64_t total_tiles,
                 const spd_stats_t *__restrict__ st, const float *__restrict__ table, int nmax,
                 float *__restrict__ snr, uint16_t *__restrict__ width,
                 int stats_stride /* 0: one spd_stats_t (and table) for all rows; 1: one per DM row */)
{
    constexpr int SW_SUB = SW_THREADS * SW_R, SW_TILE = 2 * SW_SUB;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const SweepSmem lay(nmax, SW_THREADS);
    float2 *Z   = reinterpret_cast<float2 *>(smem_raw + lay.z);
    float  *raw = reinterpret_cast<float *>(smem_raw + lay.raw);
    float  *EA  = reinterpret_cast<float *>(smem_raw + lay.ea);       // exclusive prefix sums of y, sub-tile A, groups of 8 at 12-float pitch
    float  *EB  = reinterpret_cast<float *>(smem_raw + lay.eb);
    float2 *scan = reinterpret_cast<float2 *>(smem_raw + lay.scan);   // [2][4] per-warp totals of the tile prefix scan
    float  *rtf = reinterpret_cast<float *>(smem_raw + lay.rtf);      // r_w (the width search reads it with a per-lane index)

    const int tid = threadIdx.x;
    const int lane = tid & 31, wid = tid >> 5;
    const int nblk = sw_nblk(nmax);
    const int H = sw_halo(nmax);
    const int LRAW = SW_TILE + H;                 // raw floats per tile: x[T0 .. T0 + TILE + H)
    const int LZ = SW_SUB + H;                    // interleaved positions (a multiple of 8)
    const int nparts = (LZ + SW_SUB - 1) / SW_SUB;
    Norm norm(st);
    const float NINF = __int_as_float(0xff800000);
    const int mask7 = opaque_reg(~7);
    const bool row_tables = !RC && stats_stride != 0;
    // every row of both planes 16-byte aligned: whole tiles take the straight-line store path
    const bool planes_fast = ((reinterpret_cast<uintptr_t>(snr) & 15) == 0) && ((row_stride & 3) == 0) &&
                             (width == nullptr || (((reinterpret_cast<uintptr_t>(width) & 15) == 0) && ((row_stride & 7) == 0)));

    if (!row_tables) for (int w = tid; w < sw_rt_len(nmax); w += SW_THREADS) rtf[w] = RC ? c_isqrt.v[w] : __ldg(table + w);

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
        if (stats_stride) {                        // per-row statistics: this row's mu, sigma (and r_w table)
            norm.load(st + row);
            if (row_tables) {
                __syncthreads();                   // the width search of the previous tile has read rtf
                for (int w = tid; w < sw_rt_len(nmax); w += SW_THREADS) rtf[w] = __ldg(table + row * sw_rt_len(nmax) + w);
            }
        }
        stg.wait();
        __syncthreads();                           // raw tile landed; everyone is done with the previous Z / E

        // ---- per-thread state ---------------------------------------------------------------------------------------
        float2 B[SW_R], W[SW_R], bestA[SW_R], bestB[SW_R];
        int kx[SW_R], ky[SW_R];
#pragma unroll
        for (int j = 0; j < SW_R; ++j) {
            B[j] = make_float2(0.f, 0.f);
            bestA[j] = make_float2(NINF, NINF);
            kx[j] = 0; ky[j] = 0;
        }

        // ---- staging, one pass: every thread takes groups of 8 consecutive positions (part 0: its own 8 samples, whose
        //      y values stay in registers as the first window), forms y, writes the interleaved Z and the tile-local
        //      EXCLUSIVE prefix sums E[i] = y[0] + ... + y[i-1] of both sub-tiles (only the width search reads E)
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
                        load_norm_group<SW_SUB, RC>(raw, g, norm, v);
                        store_group(Z, g, v);
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
                if (act) {                                       // group g of E: off, off + v0, ..., off + v6 (v is the inclusive scan)
                    float2 e[SW_R];
                    e[0] = off;
#pragma unroll
                    for (int j = 1; j < SW_R; ++j) e[j] = __fadd2_rn(v[j - 1], off);
                    float4 *da = reinterpret_cast<float4 *>(EA + 12 * g), *db = reinterpret_cast<float4 *>(EB + 12 * g);
                    da[0] = make_float4(e[0].x, e[1].x, e[2].x, e[3].x); da[1] = make_float4(e[4].x, e[5].x, e[6].x, e[7].x);
                    db[0] = make_float4(e[0].y, e[1].y, e[2].y, e[3].y); db[1] = make_float4(e[4].y, e[5].y, e[6].y, e[7].y);
                }
            }
        }

        // ---- main loop: blocks of 8 widths, the running maximum ping-pongs between bestA and bestB ---------------------
        {
            const float2 *zp = Z + 10 * (tid + 1);               // zpad(8 tid + 8 kb + 8 + u) = 10 (tid + kb + 1) + u
            const float *rp = rtf;
            int kb = 0;
            int kbv = opaque_reg(0);      // the block index as a per-thread value for note_block: the loop counter itself stays
                                          // warp-uniform, so c_isqrt.v[8 kb + u] is loaded into a uniform register (LDCU)
            for (; kb + 2 <= nblk; kb += 2, kbv += 2) {
                sweep8<RC>(B, W, bestA, bestB, zp, rp, 8 * kb);
                note_block(bestB, bestA, kbv, kx, ky);
                sweep8<RC>(B, W, bestB, bestA, zp + 10, rp + 8, 8 * kb + 8);
                note_block(bestA, bestB, kbv + 1, kx, ky);
                zp += 20; rp += 16;
            }
            if (kb < nblk) {
                sweep8<RC>(B, W, bestA, bestB, zp, rp, 8 * kb);
                note_block(bestB, bestA, kbv, kx, ky);
#pragma unroll
                for (int j = 0; j < SW_R; ++j) bestA[j] = bestB[j];
            }
        }
        float2 (&best)[SW_R] = bestA;
        __syncthreads();                           // E (written before the main loop) is complete for every warp

        // ---- width search inside the winning block -----------------------------------------------------------------
        int wx[SW_R], wy[SW_R];
        if (width) {
            const float4 *oa = reinterpret_cast<const float4 *>(EA + 12 * tid), *ob = reinterpret_cast<const float4 *>(EB + 12 * tid);
            const float4 a0 = oa[0], a1 = oa[1], b0 = ob[0], b1 = ob[1];          // E[t] of the thread's own 8 + 8 samples
            const float pa[8] = {a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w}, pb[8] = {b0.x, b0.y, b0.z, b0.w, b1.x, b1.y, b1.z, b1.w};
            wx[0] = width_in_block<0>(EA, rtf, tid, kx[0], pa[0], mask7); wy[0] = width_in_block<0>(EB, rtf, tid, ky[0], pb[0], mask7);
            wx[1] = width_in_block<1>(EA, rtf, tid, kx[1], pa[1], mask7); wy[1] = width_in_block<1>(EB, rtf, tid, ky[1], pb[1], mask7);
            wx[2] = width_in_block<2>(EA, rtf, tid, kx[2], pa[2], mask7); wy[2] = width_in_block<2>(EB, rtf, tid, ky[2], pb[2], mask7);
            wx[3] = width_in_block<3>(EA, rtf, tid, kx[3], pa[3], mask7); wy[3] = width_in_block<3>(EB, rtf, tid, ky[3], pb[3], mask7);
            wx[4] = width_in_block<4>(EA, rtf, tid, kx[4], pa[4], mask7); wy[4] = width_in_block<4>(EB, rtf, tid, ky[4], pb[4], mask7);
            wx[5] = width_in_block<5>(EA, rtf, tid, kx[5], pa[5], mask7); wy[5] = width_in_block<5>(EB, rtf, tid, ky[5], pb[5], mask7);
            wx[6] = width_in_block<6>(EA, rtf, tid, kx[6], pa[6], mask7); wy[6] = width_in_block<6>(EB, rtf, tid, ky[6], pb[6], mask7);
            wx[7] = width_in_block<7>(EA, rtf, tid, kx[7], pa[7], mask7); wy[7] = width_in_block<7>(EB, rtf, tid, ky[7], pb[7], mask7);
        }

        // a NaN reciprocal table (LINEAR mode fed stats of another Nmax) must surface: fmaxf drops NaN operands
        if (!RC && rtf[0] != rtf[0]) {
#pragma unroll
            for (int j = 0; j < SW_R; ++j) best[j] = make_float2(rtf[0], rtf[0]);
        }

        if (planes_fast && T0 + SW_TILE <= n_t) {             // whole tile inside 16-byte aligned planes: straight-line 16-byte streaming stores
            float *oa = snr + row * row_stride + (T0 + SW_R * tid), *ob = oa + SW_SUB;
            __stcs(reinterpret_cast<float4 *>(oa), make_float4(best[0].x, best[1].x, best[2].x, best[3].x));
            __stcs(reinterpret_cast<float4 *>(oa) + 1, make_float4(best[4].x, best[5].x, best[6].x, best[7].x));
            __stcs(reinterpret_cast<float4 *>(ob), make_float4(best[0].y, best[1].y, best[2].y, best[3].y));
            __stcs(reinterpret_cast<float4 *>(ob) + 1, make_float4(best[4].y, best[5].y, best[6].y, best[7].y));
            if (width) {
                uint16_t *wa = width + row * row_stride + (T0 + SW_R * tid), *wb = wa + SW_SUB;
                __stcs(reinterpret_cast<uint4 *>(wa), make_uint4(wx[0] | (wx[1] << 16), wx[2] | (wx[3] << 16), wx[4] | (wx[5] << 16), wx[6] | (wx[7] << 16)));
                __stcs(reinterpret_cast<uint4 *>(wb), make_uint4(wy[0] | (wy[1] << 16), wy[2] | (wy[3] << 16), wy[4] | (wy[5] << 16), wy[6] | (wy[7] << 16)));
            }
        } else {
            store_planes<SW_THREADS>(snr, width, row, row_stride, n_t, T0 + SW_R * tid, best, wx, wy);
        }
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

template <int SW_THREADS, bool RC>
__global__ void __launch_bounds__(SW_THREADS, 512 / SW_THREADS)
boxcar_search_fused(const float *__restrict__ x, int64_t n_t, int64_t row_stride, int tiles_per_row, int64_t total_tiles,
                    const spd_stats_t *__restrict__ st, const float *__restrict__ table, int nmax,
                    float threshold, spd_candidate_t *__restrict__ cand, unsigned long long capacity,
                    unsigned long long *__restrict__ count, int stats_stride)
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
    Norm norm(st);
    const float NINF = __int_as_float(0xff800000);
    const bool row_tables = !RC && stats_stride != 0;

    if (!row_tables) for (int w = tid; w < sw_rt_len(nmax); w += SW_THREADS) rtf[w] = RC ? c_isqrt.v[w] : __ldg(table + w);
    // a NaN reciprocal table (LINEAR mode fed stats of another Nmax): NaN >= threshold is false everywhere, which would
    // read as "no detections"; report the misuse as count = ~0 instead (spd.h)
    if (!RC && blockIdx.x == 0 && tid == 0) { const float r0 = __ldg(table); if (r0 != r0) *count = ~0ULL; }

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
        if (stats_stride) {
            norm.load(st + row);
            if (row_tables) {
                __syncthreads();                   // the replays of the previous tile have read rtf
                for (int w = tid; w < sw_rt_len(nmax); w += SW_THREADS) rtf[w] = __ldg(table + row * sw_rt_len(nmax) + w);
            }
        }
        stg.wait();
        __syncthreads();                           // raw tile landed; everyone is done with the previous Z

        float2 B[SW_R], W[SW_R], best[SW_R];
        load_norm_group<SW_SUB, RC>(raw, tid, norm, W);          // the thread's own 8 + 8 samples stay in registers as the first window
        store_group(Z, tid, W);
        for (int g = SW_THREADS + tid; 8 * g < LZ; g += SW_THREADS) {      // the halo positions past the sub-tile
            float2 v[SW_R];
            load_norm_group<SW_SUB, RC>(raw, g, norm, v);
            store_group(Z, g, v);
        }
        __syncthreads();                           // Z complete; raw is free again
        if (tile + gridDim.x < total_tiles) stg.stage<SW_THREADS, false>(raw, x, n_t, row_stride, pos, LRAW, tid);

#pragma unroll
        for (int j = 0; j < SW_R; ++j) { B[j] = make_float2(0.f, 0.f); best[j] = make_float2(NINF, NINF); }
        {
            const float2 *zp = Z + 10 * (tid + 1);
            const float *rp = rtf;
            int kb = 0;
            for (; kb + 2 <= nblk; kb += 2, zp += 20, rp += 16) {
                sweep8<RC>(B, W, best, best, zp, rp, 8 * kb);
                sweep8<RC>(B, W, best, best, zp + 10, rp + 8, 8 * kb + 8);
            }
            if (kb < nblk) sweep8<RC>(B, W, best, best, zp, rp, 8 * kb);
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
// One level of the FUSED decimated search (spd_search_fused_decimated; PAPER.md:97 + :87-93, reading A20): the width loop
// of boxcar_search_fused on the decimated series x_l for the level's widths w' = wmin + 1 .. nmax (nmax = w0 <= 32; the
// widths up to wmin, a multiple of 8, are only summed: they belong to the finer levels), threshold in the kernel, no
// planes.  A hit becomes the record (row, t = i wscale, snr, width = w' wscale), wscale = 2^l.  Like the narrow plane
// kernel of a level it also writes the next level's series, x_{l+1}[i] = x_l[2i] + x_l[2i+1], from the tile it has staged.
__device__ __forceinline__ void sum8(float2 (&B)[SW_R], float2 (&W)[SW_R], const float2 *__restrict__ zp)
{
#pragma unroll
    for (int u = 0; u < 8; u += 2) {
        const float4 nq = *reinterpret_cast<const float4 *>(zp + u);
        const float2 n0 = make_float2(nq.x, nq.y), n1 = make_float2(nq.z, nq.w);
#pragma unroll
        for (int j = 0; j < SW_R; ++j) {
            B[j] = __fadd2_rn(B[j], W[(j + u) & 7]);
            B[j] = __fadd2_rn(B[j], (j == SW_R - 1) ? n0 : W[(j + u + 1) & 7]);
        }
        W[u] = n0;
        W[u + 1] = n1;
    }
}

__device__ __noinline__ int replay_width_level(const float *__restrict__ zh, int pos, const float *__restrict__ rtf, int nmax, int wmin, float best)
{
    float b = 0.f;
    for (int w = 1; w <= nmax; ++w) {
        b = __fadd_rn(b, zh[2 * zpad(pos + w - 1)]);
        if (w > wmin && __fmul_rn(b, rtf[w - 1]) == best) return w;
    }
    return nmax;                                   // not reached for finite input
}

template <int SW_THREADS, bool RC, int W0, bool LEVEL0>
__global__ void __launch_bounds__(SW_THREADS, 640 / SW_THREADS)
boxcar_search_fused_level(const float *__restrict__ x, int64_t n_t, int64_t row_stride, int tiles_per_row, int64_t total_tiles,
                          const spd_stats_t *__restrict__ st, const float *__restrict__ table, int nmax, int wmin, int wscale,
                          float threshold, spd_candidate_t *__restrict__ cand, unsigned long long capacity,
                          unsigned long long *__restrict__ count, float *__restrict__ dec_out, int64_t dec_stride)
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
    const Norm norm(st);
    const float NINF = __int_as_float(0xff800000);

    for (int w = tid; w < sw_rt_len(nmax); w += SW_THREADS) rtf[w] = RC ? c_isqrt.v[w] : __ldg(table + w);
    // a NaN reciprocal table (LINEAR mode fed stats of another Nmax) is reported as count = ~0 (spd.h), as in boxcar_search_fused
    if (!RC && blockIdx.x == 0 && tid == 0) { const float r0 = __ldg(table); if (r0 != r0) *count = ~0ULL; }

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

        float2 B[SW_R], W[SW_R], best[SW_R];
        if (dec_out == nullptr) load_norm_group<SW_SUB, RC>(raw, tid, norm, W);
        else {                                     // the thread's own samples, summed in pairs: the next level's series
            float4 sa, sb;
            load_norm_group<SW_SUB, RC, true>(raw, tid, norm, W, &sa, &sb);
            const int64_t n_next = n_t >> 1;
            const int64_t ia = (T0 + SW_R * tid) >> 1, ib = ia + SW_SUB / 2;
            float *da = dec_out + row * dec_stride + ia, *db = dec_out + row * dec_stride + ib;
            const bool al = ((reinterpret_cast<uintptr_t>(dec_out + row * dec_stride) & 15) == 0);
            if (al && ia + 3 < n_next) *reinterpret_cast<float4 *>(da) = sa;
            else { const float t[4] = {sa.x, sa.y, sa.z, sa.w}; for (int k = 0; k < 4; ++k) if (ia + k < n_next) da[k] = t[k]; }
            if (al && ib + 3 < n_next) *reinterpret_cast<float4 *>(db) = sb;
            else { const float t[4] = {sb.x, sb.y, sb.z, sb.w}; for (int k = 0; k < 4; ++k) if (ib + k < n_next) db[k] = t[k]; }
        }
        store_group(Z, tid, W);
        for (int g = SW_THREADS + tid; 8 * g < LZ; g += SW_THREADS) {      // the halo positions past the sub-tile
            float2 v[SW_R];
            load_norm_group<SW_SUB, RC>(raw, g, norm, v);
            store_group(Z, g, v);
        }
        __syncthreads();                           // Z complete; raw is free again
        if (tile + gridDim.x < total_tiles) stg.stage<SW_THREADS, true>(raw, x, n_t, row_stride, pos, LRAW, tid);

#pragma unroll
        for (int j = 0; j < SW_R; ++j) { B[j] = make_float2(0.f, 0.f); best[j] = make_float2(NINF, NINF); }
        {
            // W0 and the level kind are compile-time: straight-line blocks, r_w of eq. 4 at constant offsets of the constant bank
            const float2 *zp = Z + 10 * (tid + 1);
            constexpr int NB = W0 / 8, FIRST = LEVEL0 ? 0 : NB / 2;      // blocks below FIRST are only summed (wmin = W0 / 2)
#pragma unroll
            for (int kb = 0; kb < NB; ++kb) {
                if (kb < FIRST) sum8(B, W, zp + 10 * kb);
                else sweep8<RC>(B, W, best, best, zp + 10 * kb, rtf + 8 * kb, 8 * kb);
            }
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
                if (ha) wa = replay_width_level(zf, SW_R * tid + j, rtf, nmax, wmin, best[j].x);
                if (hb) wb = replay_width_level(zf + 1, SW_R * tid + j, rtf, nmax, wmin, best[j].y);
                __syncwarp();
                append_candidate(ha, (uint32_t)row, (uint32_t)((ta + j) * wscale), best[j].x, (uint32_t)(wa * wscale), cand, capacity, count);
                append_candidate(hb, (uint32_t)row, (uint32_t)((tb + j) * wscale), best[j].y, (uint32_t)(wb * wscale), cand, capacity, count);
            }
        }
    }
    cp_async_commit_wait_all();
}

// ---------------------------------------------------------------------------------------------------------------
// Narrow searches (nmax <= SW_NARROW_NMAX = 32, the room of a 5-bit tag): the fixed per-sample cost of the general
// kernel (prefix scan + width search) is larger than the width loop itself, so here the arg-max rides along with the
// maximum: beside the exact running maximum a second one is kept over TAGGED values, (bits(s) & ~31) | (32 - w), one
// LOP3 per value.  A larger tag is a smaller width, so exact ties keep the smallest width (A7) for non-negative maxima;
// values closer than 32 ulp (4e-6 relative, far inside the 1e-3 tie tolerance of DESIGN.md section 5) may resolve
// either way.  The SNR written is the exact maximum.  A tagged -inf (a window past the row end) or NaN (a width past
// nmax) is a NaN, which FMNMX drops.  No scan, no width search, no bookkeeping.
template <int KB, bool RC, bool EVAL>
__device__ __forceinline__ void sweep8_tagged(float2 (&B)[SW_R], float2 (&W)[SW_R], float2 (&best)[SW_R], float2 (&tbest)[SW_R],
                                              const float2 *__restrict__ zp, const float *__restrict__ rp, int mask)
{
#pragma unroll
    for (int u = 0; u < 8; u += 2) {
        float2 rr;
        if (RC) rr = make_float2(c_isqrt.v[8 * KB + u], c_isqrt.v[8 * KB + u + 1]);
        else rr = *reinterpret_cast<const float2 *>(rp + u);
        const float2 r0 = make_float2(rr.x, rr.x), r1 = make_float2(rr.y, rr.y);
        const float4 nq = *reinterpret_cast<const float4 *>(zp + u);     // two window elements per 16-byte load
        const float2 n0 = make_float2(nq.x, nq.y), n1 = make_float2(nq.z, nq.w);
        const int c0 = 32 - (8 * KB + u + 1), c1 = c0 - 1;              // 32 - w for the two widths of this step
#pragma unroll
        for (int j = 0; j < SW_R; ++j) {
            B[j] = __fadd2_rn(B[j], W[(j + u) & 7]);
            const float2 s0 = __fmul2_rn(B[j], r0);
            B[j] = __fadd2_rn(B[j], (j == SW_R - 1) ? n0 : W[(j + u + 1) & 7]);
            if (!EVAL) continue;                   // a decimated level leaves its narrow widths to the finer levels: running sums only
            const float2 s1 = __fmul2_rn(B[j], r1);
            best[j].x = fmax3(best[j].x, s0.x, s1.x);
            best[j].y = fmax3(best[j].y, s0.y, s1.y);
            tbest[j].x = fmax3(tbest[j].x, tag_bits(s0.x, mask, c0), tag_bits(s1.x, mask, c1));
            tbest[j].y = fmax3(tbest[j].y, tag_bits(s0.y, mask, c0), tag_bits(s1.y, mask, c1));
        }
        W[u] = n0;
        W[u + 1] = n1;
    }
}

template <int SW_THREADS, bool RC, bool DEC>
__global__ void __launch_bounds__(SW_THREADS, 640 / SW_THREADS)
boxcar_snr_sweep_narrow(const float *__restrict__ x, int64_t n_t, int64_t row_stride, int tiles_per_row, int64_t total_tiles,
                        const spd_stats_t *__restrict__ st, const float *__restrict__ table, int nmax,
                        float *__restrict__ snr, uint16_t *__restrict__ width,
                        int wmin /* widths <= wmin are summed but not evaluated (0 or a multiple of 8) */,
                        int wscale /* reported width = w * wscale */, int64_t out_stride /* row stride of the planes */,
                        int stats_stride,
                        float *__restrict__ dec_out /* may be NULL: the next decimated level, x'[i] = x[2i] + x[2i+1] */,
                        int64_t dec_stride)
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
    Norm norm(st);
    const float NINF = __int_as_float(0xff800000);
    const int mask31 = opaque_reg(~31);
    // every row of both planes 16-byte aligned: whole tiles take the straight-line store path
    const bool planes_fast = ((reinterpret_cast<uintptr_t>(snr) & 15) == 0) && ((out_stride & 3) == 0) &&
                             (width == nullptr || (((reinterpret_cast<uintptr_t>(width) & 15) == 0) && ((out_stride & 7) == 0)));
    const bool row_tables = !RC && stats_stride != 0;

    if (!RC && !row_tables) for (int w = tid; w < sw_rt_len(nmax); w += SW_THREADS) rtf[w] = __ldg(table + w);

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
        if (stats_stride) {
            norm.load(st + row);
            if (row_tables) {
                __syncthreads();                   // the width loop of the previous tile has read rtf
                for (int w = tid; w < sw_rt_len(nmax); w += SW_THREADS) rtf[w] = __ldg(table + row * sw_rt_len(nmax) + w);
            }
        }
        stg.wait();
        __syncthreads();                           // raw tile landed; everyone is done with the previous Z

        float2 B[SW_R], W[SW_R], best[SW_R], tbest[SW_R];
        {   // the thread's own 8 + 8 samples: they stay in registers as the first window
            if (!DEC || dec_out == nullptr) load_norm_group<SW_SUB, RC>(raw, tid, norm, W);
            else {                                     // ... and, summed in pairs, they are the next level's series
                float4 sa, sb;
                load_norm_group<SW_SUB, RC, true>(raw, tid, norm, W, &sa, &sb);
                const int64_t n_next = n_t >> 1;
                const int64_t ia = (T0 + SW_R * tid) >> 1, ib = ia + SW_SUB / 2;
                float *da = dec_out + row * dec_stride + ia, *db = dec_out + row * dec_stride + ib;
                const bool al = ((reinterpret_cast<uintptr_t>(dec_out + row * dec_stride) & 15) == 0);
                if (al && ia + 3 < n_next) *reinterpret_cast<float4 *>(da) = sa;
                else { const float t[4] = {sa.x, sa.y, sa.z, sa.w}; for (int k = 0; k < 4; ++k) if (ia + k < n_next) da[k] = t[k]; }
                if (al && ib + 3 < n_next) *reinterpret_cast<float4 *>(db) = sb;
                else { const float t[4] = {sb.x, sb.y, sb.z, sb.w}; for (int k = 0; k < 4; ++k) if (ib + k < n_next) db[k] = t[k]; }
            }
            store_group(Z, tid, W);
        }
        for (int g = SW_THREADS + tid; 8 * g < LZ; g += SW_THREADS) {      // the halo positions past the sub-tile
            float2 v[SW_R];
            load_norm_group<SW_SUB, RC>(raw, g, norm, v);
            store_group(Z, g, v);
        }
        __syncthreads();                           // Z complete; raw is free again
        if (tile + gridDim.x < total_tiles) stg.stage<SW_THREADS, true>(raw, x, n_t, row_stride, pos, LRAW, tid);

#pragma unroll
        for (int j = 0; j < SW_R; ++j) { B[j] = make_float2(0.f, 0.f); best[j] = make_float2(NINF, NINF); tbest[j] = make_float2(NINF, NINF); }
        const float2 *zp = Z + 10 * (tid + 1);
        if (wmin >= 8) sweep8_tagged<0, RC, false>(B, W, best, tbest, zp, rtf, mask31);
        else sweep8_tagged<0, RC, true>(B, W, best, tbest, zp, rtf, mask31);
        if (nblk > 1) {
            if (wmin >= 16) sweep8_tagged<1, RC, false>(B, W, best, tbest, zp + 10, rtf + 8, mask31);
            else sweep8_tagged<1, RC, true>(B, W, best, tbest, zp + 10, rtf + 8, mask31);
        }
        if (nblk > 2) sweep8_tagged<2, RC, true>(B, W, best, tbest, zp + 20, rtf + 16, mask31);
        if (nblk > 3) sweep8_tagged<3, RC, true>(B, W, best, tbest, zp + 30, rtf + 24, mask31);

        if (planes_fast && T0 + SW_TILE + (DEC ? H : 0) <= n_t && (RC || rtf[0] == rtf[0])) {      // (a NaN table must surface: general path;
                                                               //  a decimated level: every width must fit at every position of the tile)
            // whole tile inside 16-byte aligned planes (all but the last tile of a row): six 16-byte streaming stores per thread,
            // and the widths are decoded two at a time, (32 - tag_lo) | (32 - tag_hi) << 16 = 0x00200020 - (tags picked by PRMT)
            float *oa = snr + row * out_stride + (T0 + SW_R * tid), *ob = oa + SW_SUB;
            __stcs(reinterpret_cast<float4 *>(oa), make_float4(best[0].x, best[1].x, best[2].x, best[3].x));
            __stcs(reinterpret_cast<float4 *>(oa) + 1, make_float4(best[4].x, best[5].x, best[6].x, best[7].x));
            __stcs(reinterpret_cast<float4 *>(ob), make_float4(best[0].y, best[1].y, best[2].y, best[3].y));
            __stcs(reinterpret_cast<float4 *>(ob) + 1, make_float4(best[4].y, best[5].y, best[6].y, best[7].y));
            if (width) {
                uint16_t *wa = width + row * out_stride + (T0 + SW_R * tid), *wb = wa + SW_SUB;
                unsigned pa[4], pb[4];
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    pa[k] = 0x00200020u - (__byte_perm(__float_as_uint(tbest[2 * k].x), __float_as_uint(tbest[2 * k + 1].x), 0x4400) & 0x001f001fu);
                    pb[k] = 0x00200020u - (__byte_perm(__float_as_uint(tbest[2 * k].y), __float_as_uint(tbest[2 * k + 1].y), 0x4400) & 0x001f001fu);
                    if (DEC) { pa[k] *= (unsigned)wscale; pb[k] *= (unsigned)wscale; }       // effective widths w' 2^l <= 4096: no carry between the halves
                }
                __stcs(reinterpret_cast<uint4 *>(wa), make_uint4(pa[0], pa[1], pa[2], pa[3]));
                __stcs(reinterpret_cast<uint4 *>(wb), make_uint4(pb[0], pb[1], pb[2], pb[3]));
            }
            continue;
        }

        int wx[SW_R], wy[SW_R];
#pragma unroll
        for (int j = 0; j < SW_R; ++j) {
            wx[j] = (32 - (__float_as_int(tbest[j].x) & 31)) * wscale; wy[j] = (32 - (__float_as_int(tbest[j].y) & 31)) * wscale;
            if (wmin > 0) {                         // a position where none of the level's widths fits: snr = -inf, width = 0
                if (best[j].x == NINF) wx[j] = 0;
                if (best[j].y == NINF) wy[j] = 0;
            }
        }
        if (!RC && rtf[0] != rtf[0]) {              // NaN table (LINEAR mode fed stats of another Nmax) must surface
#pragma unroll
            for (int j = 0; j < SW_R; ++j) { best[j] = make_float2(rtf[0], rtf[0]); wx[j] = 1; wy[j] = 1; }
        }
        store_planes<SW_THREADS>(snr, width, row, out_stride, n_t, T0 + SW_R * tid, best, wx, wy);
    }
    cp_async_commit_wait_all();
}

// ---- launch: one resident wave of persistent CTAs.  The occupancy of a (kernel, shared-memory size, device) is looked up
// once and cached, and the kernel's dynamic shared-memory limit is only ever raised (the queries cost ~40 us per launch
// otherwise; config 1 is launch-latency-bound).
struct GridCache {
    std::mutex mu;
    struct Entry { const void *fn; int smem, dev, ctas; };
    Entry e[256];
    int n = 0;
    int limit(const void *fn, int dev) const          // largest dynamic shared-memory size set for this kernel so far
    {
        int m = 0;
        for (int i = 0; i < n; ++i) if (e[i].fn == fn && e[i].dev == dev && e[i].smem > m) m = e[i].smem;
        return m;
    }
};
static GridCache g_grid_cache;

template <typename K>
static cudaError_t persistent_grid(K kernel, int threads, int smem, int64_t tiles, unsigned *grid)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    const void *fn = reinterpret_cast<const void *>(kernel);
    int wave = 0;
    {
        std::lock_guard<std::mutex> lk(g_grid_cache.mu);
        for (int i = 0; i < g_grid_cache.n; ++i) {
            const GridCache::Entry &c = g_grid_cache.e[i];
            if (c.fn == fn && c.smem == smem && c.dev == dev) { wave = c.ctas; break; }
        }
        if (wave == 0) {
            int sms = 0, per_sm = 0;
            const bool full = g_grid_cache.n >= 256;             // table full: set the attribute every time, never below a cached size
            const int lim = g_grid_cache.limit(fn, dev);
            if (full || smem > lim)
                if ((e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem > lim ? smem : lim)) != cudaSuccess) return e;
            if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
            if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, threads, smem)) != cudaSuccess) return e;
            if (per_sm < 1) return cudaErrorInvalidConfiguration;
            wave = sms * per_sm;                                 // persistent: one resident wave walks all tiles
            if (!full) g_grid_cache.e[g_grid_cache.n++] = GridCache::Entry{fn, smem, dev, wave};
        }
    }
    *grid = (unsigned)(tiles < wave ? tiles : (int64_t)wave);
    return cudaSuccess;
}

template <int NT, bool RC>
static cudaError_t launch_sweep_nt(const float *x, int64_t n_dm, int64_t n_t, int64_t row_stride, const spd_stats_t *d_stats,
                                   const float *d_table, int nmax, float *snr, uint16_t *width,
                                   bool fused, float threshold, spd_candidate_t *out, unsigned long long capacity,
                                   unsigned long long *d_count, cudaStream_t s, int stats_stride)
{
    constexpr int TILE = 2 * NT * SW_R;
    const int tpr = (int)((n_t + TILE - 1) / TILE);
    const int64_t tiles = n_dm * (int64_t)tpr;
    unsigned grid = 0;
    cudaError_t e;
    if constexpr (NT == 32) {                      // one-warp CTAs: the general plane kernel only
        const SweepSmem lay(nmax, NT);
        if ((e = persistent_grid(boxcar_snr_sweep<NT, RC>, NT, lay.total, tiles, &grid)) != cudaSuccess) return e;
        boxcar_snr_sweep<NT, RC><<<grid, NT, lay.total, s>>>(x, n_t, row_stride, tpr, tiles, d_stats, d_table, nmax, snr, width, stats_stride);
    } else if (fused) {
        const FusedSmem lay(nmax, NT);
        if ((e = persistent_grid(boxcar_search_fused<NT, RC>, NT, lay.total, tiles, &grid)) != cudaSuccess) return e;
        boxcar_search_fused<NT, RC><<<grid, NT, lay.total, s>>>(x, n_t, row_stride, tpr, tiles, d_stats, d_table, nmax,
                                                                threshold, out, capacity, d_count, stats_stride);
    } else if (nmax <= SW_NARROW_NMAX) {
        const FusedSmem lay(nmax, NT);
        if ((e = persistent_grid(boxcar_snr_sweep_narrow<NT, RC, false>, NT, lay.total, tiles, &grid)) != cudaSuccess) return e;
        boxcar_snr_sweep_narrow<NT, RC, false><<<grid, NT, lay.total, s>>>(x, n_t, row_stride, tpr, tiles, d_stats, d_table, nmax, snr, width,
                                                                    0, 1, row_stride, stats_stride, nullptr, 0);
    } else {
        const SweepSmem lay(nmax, NT);
        if ((e = persistent_grid(boxcar_snr_sweep<NT, RC>, NT, lay.total, tiles, &grid)) != cudaSuccess) return e;
        boxcar_snr_sweep<NT, RC><<<grid, NT, lay.total, s>>>(x, n_t, row_stride, tpr, tiles, d_stats, d_table, nmax, snr, width, stats_stride);
    }
    return cudaGetLastError();
}

// rc = sweep_uses_constant_table(nmax, mode): eq. 4 with nmax a multiple of 8 (d_table is then not read)
cudaError_t launch_sweep(const float *x, int64_t n_dm, int64_t n_t, int64_t row_stride, const spd_stats_t *d_stats,
                         const float *d_table, int nmax, bool rc, float *snr, uint16_t *width,
                         bool fused, float threshold, spd_candidate_t *out, unsigned long long capacity,
                         unsigned long long *d_count, cudaStream_t s, int stats_stride)
{
    if (fused && stats_stride == 0 && nmax <= 32 && (nmax & 7) == 0)        // narrow fused search: the straight-line level kernel (level 0, scale 1)
        return launch_search_level(x, n_dm, n_t, row_stride, d_stats, d_table, nmax, 0, 1, rc, threshold, out, capacity, d_count, nullptr, 0, s);
    if (!fused && nmax > SW_NARROW_NMAX && nmax <= SW_WARP_CTA_NMAX) {       // general plane kernel, one-warp CTAs
        if (rc) return launch_sweep_nt<32, true>(x, n_dm, n_t, row_stride, d_stats, d_table, nmax, snr, width, fused, threshold, out, capacity, d_count, s, stats_stride);
        return launch_sweep_nt<32, false>(x, n_dm, n_t, row_stride, d_stats, d_table, nmax, snr, width, fused, threshold, out, capacity, d_count, s, stats_stride);
    }
    if (nmax <= SW_SMALL_CTA_NMAX) {
        if (rc) return launch_sweep_nt<64, true>(x, n_dm, n_t, row_stride, d_stats, d_table, nmax, snr, width, fused, threshold, out, capacity, d_count, s, stats_stride);
        return launch_sweep_nt<64, false>(x, n_dm, n_t, row_stride, d_stats, d_table, nmax, snr, width, fused, threshold, out, capacity, d_count, s, stats_stride);
    }
    if (rc) return launch_sweep_nt<128, true>(x, n_dm, n_t, row_stride, d_stats, d_table, nmax, snr, width, fused, threshold, out, capacity, d_count, s, stats_stride);
    return launch_sweep_nt<128, false>(x, n_dm, n_t, row_stride, d_stats, d_table, nmax, snr, width, fused, threshold, out, capacity, d_count, s, stats_stride);
}

// one level of the decimated search: the narrow kernel on the decimated series x_l (w0 <= 32) with the level's statistics
cudaError_t launch_sweep_level(const float *xl, int64_t n_dm, int64_t n_l, int64_t xl_stride, const spd_stats_t *d_stats_level,
                               const float *d_table, int w0, int wmin, int wscale, bool rc, float *snr, uint16_t *width,
                               int64_t out_stride, float *dec_out, int64_t dec_stride, cudaStream_t s)
{
    constexpr int NT = 64, TILE = 2 * NT * SW_R;
    if (n_l <= 0) return cudaSuccess;
    const int tpr = (int)((n_l + TILE - 1) / TILE);
    const int64_t tiles = n_dm * (int64_t)tpr;
    const FusedSmem lay(w0, NT);
    unsigned grid = 0;
    cudaError_t e;
    if (rc) {
        if ((e = persistent_grid(boxcar_snr_sweep_narrow<NT, true, true>, NT, lay.total, tiles, &grid)) != cudaSuccess) return e;
        boxcar_snr_sweep_narrow<NT, true, true><<<grid, NT, lay.total, s>>>(xl, n_l, xl_stride, tpr, tiles, d_stats_level, d_table, w0, snr, width, wmin, wscale, out_stride, 0, dec_out, dec_stride);
    } else {
        if ((e = persistent_grid(boxcar_snr_sweep_narrow<NT, false, true>, NT, lay.total, tiles, &grid)) != cudaSuccess) return e;
        boxcar_snr_sweep_narrow<NT, false, true><<<grid, NT, lay.total, s>>>(xl, n_l, xl_stride, tpr, tiles, d_stats_level, d_table, w0, snr, width, wmin, wscale, out_stride, 0, dec_out, dec_stride);
    }
    return cudaGetLastError();
}

template <bool RC, int W0, bool LEVEL0>
static cudaError_t launch_search_level_t(const float *xl, int64_t n_dm, int64_t n_l, int64_t xl_stride, const spd_stats_t *d_stats_level,
                                         const float *d_table, int wscale, float threshold, spd_candidate_t *out,
                                         unsigned long long capacity, unsigned long long *d_count, float *dec_out, int64_t dec_stride, cudaStream_t s)
{
    constexpr int NT = 64, TILE = 2 * NT * SW_R;
    const int tpr = (int)((n_l + TILE - 1) / TILE);
    const int64_t tiles = n_dm * (int64_t)tpr;
    const FusedSmem lay(W0, NT);
    unsigned grid = 0;
    cudaError_t e;
    if ((e = persistent_grid(boxcar_search_fused_level<NT, RC, W0, LEVEL0>, NT, lay.total, tiles, &grid)) != cudaSuccess) return e;
    boxcar_search_fused_level<NT, RC, W0, LEVEL0><<<grid, NT, lay.total, s>>>(xl, n_l, xl_stride, tpr, tiles, d_stats_level, d_table, W0,
                                                                              LEVEL0 ? 0 : W0 / 2, wscale, threshold, out, capacity, d_count,
                                                                              dec_out, dec_stride);
    return cudaGetLastError();
}

// one level of the fused decimated search (w0 = 16 or 32; wmin = 0 at level 0, w0 / 2 above): threshold in the kernel, hits
// appended to one list for all levels
cudaError_t launch_search_level(const float *xl, int64_t n_dm, int64_t n_l, int64_t xl_stride, const spd_stats_t *d_stats_level,
                                const float *d_table, int w0, int wmin, int wscale, bool rc, float threshold, spd_candidate_t *out,
                                unsigned long long capacity, unsigned long long *d_count, float *dec_out, int64_t dec_stride, cudaStream_t s)
{
    if (n_l <= 0) return cudaSuccess;
    if (w0 < 8 || w0 > 32 || (w0 & 7) || (wmin != 0 && (wmin != w0 / 2 || (w0 & 15)))) return cudaErrorInvalidValue;
#define SPD_LEVEL(RC_, W0_, L0_) launch_search_level_t<RC_, W0_, L0_>(xl, n_dm, n_l, xl_stride, d_stats_level, d_table, wscale, threshold, out, capacity, d_count, dec_out, dec_stride, s)
    if (w0 == 8) return rc ? SPD_LEVEL(true, 8, true) : SPD_LEVEL(false, 8, true);            // (exhaustive fused search at Nmax 8 / 24)
    if (w0 == 24) return rc ? SPD_LEVEL(true, 24, true) : SPD_LEVEL(false, 24, true);
    if (w0 == 16) {
        if (wmin == 0) return rc ? SPD_LEVEL(true, 16, true) : SPD_LEVEL(false, 16, true);
        return rc ? SPD_LEVEL(true, 16, false) : SPD_LEVEL(false, 16, false);
    }
    if (wmin == 0) return rc ? SPD_LEVEL(true, 32, true) : SPD_LEVEL(false, 32, true);
    return rc ? SPD_LEVEL(true, 32, false) : SPD_LEVEL(false, 32, false);
#undef SPD_LEVEL
}

}  // namespace spd
