// stats.cu -- step 1 of the path: mean and standard deviation (section 2.1), and the "true"
// sigma_Nmax of eq. 5 (section 2.2) IN THE SAME PASS over x.
//
// Kernel 1: the array is cut into equal chunks of 4096 samples; every thread runs the streaming update eq. 1 over a
// fixed run of 16 samples (division-free: 1/(j(j-1)) are compile-time constants), the 32 runs of a warp are merged
// pairwise with eq. 2 through shuffles, and the warp's 512-sample partial is merged (eq. 2, fp64) into a per-warp
// accumulator.  Each CTA writes one (m, T, S) partial.  Two variants:
//   stats_partial      (nmax_for_sigma = 0): 16-byte streaming loads straight into registers.
//   stats_partial_win  (nmax_for_sigma > 0): the chunk and its nmax-1 halo samples are staged in shared memory ONCE;
//                      the same data gives the sample statistics (eq. 1 per 16-sample run, eq. 2 into a per-lane partial
//                      that lives across tiles) and the Nmax-sample boxcar SUMS of every full window: the first window
//                      of a thread from an exclusive scan over the 16-sample RUN TOTALS of the tile (by-products of
//                      eq. 1), the next 15 by sliding; their statistics are sums of b and b^2 about the shift (the paper
//                      prescribes no method for sigma_Nmax).  x is read once (plus the halo, which hits L2).
// Kernel 2 (stats_finalize) merges the partials with eq. 2 in index order (fp64, fixed order => bit-reproducible) and
// writes mu = T/n, sigma = sqrt(S/n), sigma_nmax.
//
// Precision (reading A4): fp32 inside a warp-chunk (<= 512 values), fp64 above it.  All samples are shifted
// by a per-CTA constant K before they enter eq. 1 (eq. 1/2 are applied to x - K; S is shift-invariant and T is
// un-shifted in fp64 when the CTA writes its partial), which keeps fp32 accurate when |mu| >> sigma.  K is the MEAN of
// the first chunk the CTA works on, so one outlier sample cannot spoil it.
//
// Roofline: pure HBM stream, 4 B/sample read.
#include "spd_common.cuh"

#include <mutex>

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

// eq. 1 over a full run of 16 values
__device__ __forceinline__ void chan_run16(const float (&v)[ST_RUN], float &T, float &S)
{
    T = v[0]; S = 0.0f;
    chan_push<2>(T, S, v[1]);   chan_push<3>(T, S, v[2]);   chan_push<4>(T, S, v[3]);   chan_push<5>(T, S, v[4]);
    chan_push<6>(T, S, v[5]);   chan_push<7>(T, S, v[6]);   chan_push<8>(T, S, v[7]);   chan_push<9>(T, S, v[8]);
    chan_push<10>(T, S, v[9]);  chan_push<11>(T, S, v[10]); chan_push<12>(T, S, v[11]); chan_push<13>(T, S, v[12]);
    chan_push<14>(T, S, v[13]); chan_push<15>(T, S, v[14]); chan_push<16>(T, S, v[15]);
}

// eq. 2 for two partials of EQUAL size m: S = S1 + S2 + (T1 - T2)^2 / (2m)
__device__ __forceinline__ void merge_equal(float &T, float &S, float T2, float S2, float inv_2m)
{
    float d = T - T2;
    S = fmaf(d * d, inv_2m, S + S2);
    T += T2;
}

// the 32 full runs of a warp -> one 512-value partial on every lane (eq. 2, equal sizes at each level)
__device__ __forceinline__ void warp_merge_full(float &T, float &S)
{
#pragma unroll
    for (int lvl = 0; lvl < 5; ++lvl) {
        float T2 = __shfl_xor_sync(0xffffffffu, T, 1 << lvl);
        float S2 = __shfl_xor_sync(0xffffffffu, S, 1 << lvl);
        merge_equal(T, S, T2, S2, 1.0f / (float)(2 * (ST_RUN << lvl)));
    }
}

// eq. 2 for accumulator (+) one FULL 512-value warp chunk (T, S in fp32): the hot merge, once per warp
// and tile.  Same quantity as tri_merge, (n T1 - m T2)^2 / (m n (m + n)), with the reciprocal of m n (m + n) taken in
// fp32 instead of an fp64 division (a ~60-instruction subroutine): the term is the between-chunk correction, a small
// fraction of S, so 1e-7 relative in it is orders of magnitude below the 1e-6 tolerance on sigma.
__device__ __forceinline__ void tri_merge_chunk(Tri &a, float T, float S)
{
    const double n = 512.0;
    if (a.m == 0.0) { a.m = n; a.T = (double)T; a.S = (double)S; return; }
    const double d = n * a.T - a.m * (double)T;
    const float rf = __frcp_rn((float)a.m * (float)(a.m + n));
    a.S = a.S + (double)S + d * d * ((double)rf * (1.0 / 512.0));
    a.T += (double)T;
    a.m += n;
}

// runs of any length (ragged chunk): eq. 2 in fp64, the left operand always being the lower lanes
__device__ __forceinline__ void warp_merge_ragged(Tri &t, int lane)
{
#pragma unroll
    for (int lvl = 0; lvl < 5; ++lvl) {
        Tri o;
        o.m = __shfl_xor_sync(0xffffffffu, t.m, 1 << lvl);
        o.T = __shfl_xor_sync(0xffffffffu, t.T, 1 << lvl);
        o.S = __shfl_xor_sync(0xffffffffu, t.S, 1 << lvl);
        if ((lane >> lvl) & 1) { Tri a = o; tri_merge(a, t); t = a; } else tri_merge(t, o);
    }
}

// eq. 1 with a run-time j over the first `cnt` of up to 16 values (ragged run)
__device__ __forceinline__ Tri chan_run_ragged(const float (&v)[ST_RUN], int cnt)
{
    float T = 0.0f, S = 0.0f;
    for (int k = 0; k < ST_RUN; ++k) {
        if (k < cnt) {
            if (k == 0) { T = v[0]; S = 0.0f; }
            else { T += v[k]; const float j = (float)(k + 1); const float d = fmaf(j, v[k], -T); S += d * d / (j * (j - 1.0f)); }
        }
    }
    Tri t = {(double)(cnt > 0 ? cnt : 0), (double)T, (double)S};
    if (cnt <= 0) { t.T = 0.0; t.S = 0.0; }
    return t;
}

// block-wide sum of (s, c) -> every thread gets the totals (used once per CTA for the shift K)
__device__ __forceinline__ float cta_mean(float s, float c, float *sh)
{
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) { s += __shfl_xor_sync(0xffffffffu, s, d); c += __shfl_xor_sync(0xffffffffu, c, d); }
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (lane == 0) { sh[2 * wid] = s; sh[2 * wid + 1] = c; }
    __syncthreads();
    float S = 0.f, Cn = 0.f;
#pragma unroll
    for (int w = 0; w < ST_THREADS / 32; ++w) { S += sh[2 * w]; Cn += sh[2 * w + 1]; }
    __syncthreads();
    return Cn > 0.f ? S / Cn : 0.f;
}

__device__ __forceinline__ void write_partial(Tri *warp_acc, const Tri &acc, double K, double per_value, Tri *__restrict__ out, bool per_lane = false)
{
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    Tri wa = acc;
    if (per_lane) warp_merge_ragged(wa, lane);                 // every lane holds an accumulator: fold them first (fixed order)
    if (lane == 0) warp_acc[wid] = wa;
    __syncthreads();
    if (tid == 0) {
        Tri a = warp_acc[0];
        for (int w = 1; w < ST_THREADS / 32; ++w) tri_merge(a, warp_acc[w]);
        a.T += a.m * K * per_value;                            // undo the shift: every value carried per_value * K less
        *out = a;
    }
    __syncthreads();
}

__global__ void __launch_bounds__(ST_THREADS)
stats_partial(const float *__restrict__ x, int64_t n_rows, int64_t n_t, int64_t row_stride, Tri *__restrict__ partials)
{
    // per-row statistics (spd_stats_rows): gridDim.y = rows, every y-slice is an independent one-row problem
    x += (int64_t)blockIdx.y * row_stride;
    partials += (size_t)blockIdx.y * gridDim.x;
    __shared__ Tri warp_acc[ST_THREADS / 32];
    __shared__ float red[2 * ST_THREADS / 32];
    const int tid = threadIdx.x, lane = tid & 31;
    const int64_t cpr = (n_t + ST_CHUNK - 1) / ST_CHUNK;       // chunks per row
    const int64_t total = n_rows * cpr;
    Tri acc = {0.0, 0.0, 0.0};                                 // lane 0 of each warp owns it

    // shift K of this CTA: the mean of its first chunk
    float K;
    {
        const int64_t c = blockIdx.x;
        const int64_t row = c / cpr, off = (c - row * cpr) * ST_CHUNK;
        float s = 0.f, cn = 0.f;
        for (int k = 0; k < ST_RUN; ++k) {
            const int64_t p = off + (int64_t)((k >> 2) * ST_THREADS + tid) * 4 + (k & 3);
            if (p < n_t) { s += __ldg(x + row * row_stride + p); cn += 1.f; }
        }
        K = cta_mean(s, cn, red);
    }

    // (row, chunk-in-row) advanced with 32-bit arithmetic where the chunk count allows it
    const bool small = cpr < 0x7fffffffLL;
    int64_t row = (int64_t)blockIdx.x / cpr;
    int64_t cir = (int64_t)blockIdx.x - row * cpr;
    for (int64_t c = blockIdx.x; c < total; c += gridDim.x) {
        const int64_t off = cir * ST_CHUNK;
        const int64_t row_now = row;
        if (small) {
            unsigned t = (unsigned)cir + gridDim.x;
            if (t >= (unsigned)cpr) { const unsigned q = t / (unsigned)cpr; row += q; t -= q * (unsigned)cpr; }
            cir = t;
        } else { const int64_t cn = c + gridDim.x; row = cn / cpr; cir = cn - row * cpr; }
        const float *base = x + row_now * row_stride + off;
        const bool full = (off + ST_CHUNK <= n_t) && ((reinterpret_cast<uintptr_t>(base) & 15) == 0);
        float v[ST_RUN];
        if (full) {
            float4 q[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) q[k] = ldg_stream4(base + (k * ST_THREADS + tid) * 4);
#pragma unroll
            for (int k = 0; k < 4; ++k) { v[4 * k] = q[k].x - K; v[4 * k + 1] = q[k].y - K; v[4 * k + 2] = q[k].z - K; v[4 * k + 3] = q[k].w - K; }
            float T, S;
            chan_run16(v, T, S);
            warp_merge_full(T, S);
            if (lane == 0) tri_merge_chunk(acc, T, S);
        } else {
            // ragged / unaligned chunk: eq. 1 with a run-time j, eq. 2 merges in fp64
            int cnt = 0;
#pragma unroll
            for (int k = 0; k < ST_RUN; ++k) {                 // positions ascend with k, so the valid samples are a prefix of the run
                const int64_t p = off + (int64_t)((k >> 2) * ST_THREADS + tid) * 4 + (k & 3);
                const bool ok = p < n_t;
                v[k] = ok ? __ldg(x + row_now * row_stride + p) - K : 0.0f;
                cnt += ok ? 1 : 0;
            }
            Tri t = chan_run_ragged(v, cnt);
            warp_merge_ragged(t, lane);
            if (lane == 0) tri_merge(acc, t);
        }
    }
    write_partial(warp_acc, acc, (double)K, 1.0, partials + blockIdx.x);
}

// ---- sample statistics AND sigma_Nmax in one pass (reading A11: population std of the Nmax-sample boxcar
// SUMS over every full window of every row).  One tile = 4096 consecutive samples of one row (+ nmax-1 halo samples)
// staged in shared memory with one pad float4 per 16 floats (lane stride 80 B: conflict-free 16-byte accesses).  A
// thread owns 16 consecutive positions: its samples (eq. 1, as above) and the 16 windows that START there.  Window sums
// are tile-local: B(t0) = P[t0 + nmax] - P[t0] from an fp32 prefix scan of x - K over tile + halo (P restarts at every
// tile, so it stays small), then B(t0 + k + 1) = B(t0 + k) + x[t0 + k + nmax] - x[t0 + k].
__host__ __device__ __forceinline__ int st_pad(int i) { return i + ((i >> 4) << 2); }

__device__ __forceinline__ void cp_async16_st(void *smem, const void *gmem)
{
    unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" :: "r"(s), "l"(gmem) : "memory");
}

__device__ __forceinline__ void load16(const float *sm, int pos, float (&v)[ST_RUN])      // pos a multiple of 4
{
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const float4 q = *reinterpret_cast<const float4 *>(sm + st_pad(pos + 4 * k));
        v[4 * k] = q.x; v[4 * k + 1] = q.y; v[4 * k + 2] = q.z; v[4 * k + 3] = q.w;
    }
}

// What one lane of stats_partial_win carries from tile to tile (the lanes are merged once, when the CTA writes its partials):
//   samples : the Chan partial of its runs (eq. 1 per 16-value run, eq. 2 between runs), fp32 for up to 32 runs = 512 values
//             (m32, T32, S32), folded into the fp64 partial `acc` every 32 tiles -- the precision rule of reading A4;
//   windows : the sums of b and b^2 of its windows about the shift (b = window sum of x - K, so its mean is nmax (mu - K),
//             small against its spread), fp32 over the 16 windows of a tile, fp64 across tiles.  The paper prescribes no
//             method for sigma_Nmax; S_b = sum b^2 - (sum b)^2 / n is formed in fp64 when the lane's partial is
//             written, and everything above a lane is eq. 2 again.
struct LaneAcc {
    float m32, T32, S32;
    Tri acc;
    double sb, sb2, nb;
    __device__ __forceinline__ void init() { m32 = 0.f; T32 = 0.f; S32 = 0.f; acc = Tri{0.0, 0.0, 0.0}; sb = 0.0; sb2 = 0.0; nb = 0.0; }
    // eq. 2: (m32, T32, S32) (+) one full run (16, T, S)
    __device__ __forceinline__ void push_run(float T, float S)
    {
        if (m32 == 0.f) { m32 = (float)ST_RUN; T32 = T; S32 = S; return; }
        const float d = fmaf((float)ST_RUN, T32, -m32 * T);
        const float rf = __frcp_rn(m32 * (m32 + (float)ST_RUN)) * (1.0f / (float)ST_RUN);
        S32 = fmaf(d * d, rf, S32 + S);
        T32 += T;
        m32 += (float)ST_RUN;
        if (m32 == 512.f) { tri_merge_chunk(acc, T32, S32); m32 = 0.f; }
    }
    __device__ __forceinline__ void flush()                     // fold a pending fp32 partial (fewer than 32 runs) into acc
    {
        if (m32 > 0.f) { const Tri t = {(double)m32, (double)T32, (double)S32}; tri_merge(acc, t); m32 = 0.f; }
    }
    __device__ __forceinline__ Tri windows() const
    {
        Tri t = {nb, sb, 0.0};
        if (nb > 0.0) { t.S = sb2 - sb * sb / nb; if (t.S < 0.0) t.S = 0.0; }
        return t;
    }
};

// inclusive warp scan: the shuffle's own predicate (source lane exists) guards the add
__device__ __forceinline__ float warp_scan_incl(float v)
{
#pragma unroll
    for (int d = 1; d < 32; d <<= 1)
        asm volatile("{.reg .pred p; .reg .f32 t; shfl.sync.up.b32 t|p, %0, %1, 0, 0xffffffff; @p add.f32 %0, %0, t;}" : "+f"(v) : "r"(d));
    return v;
}

// both scans of a halo warp, level by level (two independent chains)
__device__ __forceinline__ void warp_scan_incl2(float &a, float &b)
{
#pragma unroll
    for (int d = 1; d < 32; d <<= 1)
        asm volatile("{.reg .pred p; .reg .f32 t, u; shfl.sync.up.b32 t|p, %0, %2, 0, 0xffffffff; shfl.sync.up.b32 u, %1, %2, 0, 0xffffffff;\n\t"
                     "@p add.f32 %0, %0, t; @p add.f32 %1, %1, u;}" : "+f"(a), "+f"(b) : "r"(d));
}

// split CTA barrier: an mbarrier in shared memory; arrive does not wait, wait spins on the phase parity (acquire)
__device__ __forceinline__ void mbar_init(unsigned long long *b, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"((unsigned)__cvta_generic_to_shared(b)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned long long *b)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" :: "r"((unsigned)__cvta_generic_to_shared(b)) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *b, unsigned parity)
{
    unsigned ok;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"((unsigned)__cvta_generic_to_shared(b)), "r"(parity) : "memory");
    } while (!ok);
}

// One tile of stats_partial_win.  FAST = interior tile of a 16-byte aligned row: all 4096 samples, the whole halo and all
// 4096 windows exist, so every run is full and nothing needs masking (63 of 64 tiles of a 262144-sample row).
//
// First window of a thread, B(own) with own = 16 tid: the window [own, own + nmax) is q = nmax / 16 whole thread runs
// (runs tid .. tid + q - 1; run r = positions [16 r, 16 r + 16)) plus the first rem = nmax % 16 values of run tid + q.  The
// run totals are by-products: the tile's own 256 runs give theirs to eq. 1 anyway (T of chan_run16), the q - 1 halo runs
// that are needed whole are summed by the first q - 1 threads.  One exclusive scan over those <= 511 run totals, Q[r] =
// sum of runs 0 .. r-1 of y = x - K, gives B(own) = Q[tid + q] - Q[tid] (+ the rem values): no per-sample prefix sums.
// The other 15 windows slide: B(t + 1) = B(t) + x[t + nmax] - x[t].
template <bool FAST>
__device__ __forceinline__ void win_tile(const float *__restrict__ xs, float *__restrict__ Q, float (*wtot)[ST_THREADS / 32],
                                         int64_t t0, int64_t n_t, int64_t nwin, int nmax, float K, LaneAcc &L,
                                         unsigned long long *mbar, unsigned parity)
{
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int own = ST_RUN * tid;                              // first position of this thread inside the tile
    const int q = nmax >> 4, rem = nmax & 15;
    const int nh = q > 0 ? q - 1 : 0;                          // halo runs needed whole: runs 256 .. 256 + nh - 1
    float xo[ST_RUN];
    load16(xs, own, xo);
    int cnt = ST_RUN, wcnt = ST_RUN;
    if (!FAST) {
        const int64_t left = n_t - (t0 + own), wleft = nwin - (t0 + own);
        cnt = left >= ST_RUN ? ST_RUN : (left > 0 ? (int)left : 0);      // valid samples from the thread's first position on
        wcnt = wleft >= ST_RUN ? ST_RUN : (wleft > 0 ? (int)wleft : 0);  // full windows that start there
    }

    // ---- run totals first (the other warps wait for them), then the scan; the CTA-wide steps are split barriers
    //      (arrive ... independent work ... sync), so a warp that is ahead keeps issuing ----
    float y[ST_RUN];
#pragma unroll
    for (int k = 0; k < ST_RUN; ++k) y[k] = (FAST || k < cnt) ? xo[k] - K : 0.f;
    // ---- sample statistics of the tile's own 4096 positions (eq. 1 per run, eq. 2 into the lane's partial); the run total
    //      rt = sum of y is eq. 1's own T ----
    float rt;
    if (FAST || cnt == ST_RUN) {
        float T, S;
        chan_run16(y, T, S);
        rt = T;
        L.push_run(T, S);
    } else {
        const Tri t = chan_run_ragged(y, cnt);
        rt = (float)t.T;
        L.flush();
        tri_merge(L.acc, t);
    }
    const bool hwarp = 32 * wid < nh + 1;                      // warp-uniform: this warp holds halo runs (or the entry after the last)
    float ht = 0.f;
    if (tid < nh) {                                            // thread tid sums halo run tid
        float h[ST_RUN];
        load16(xs, ST_CHUNK + own, h);
#pragma unroll
        for (int k = 0; k < ST_RUN; ++k) ht += (FAST || t0 + ST_CHUNK + own + k < n_t) ? h[k] - K : 0.f;
    }
    float inc = rt, inch = ht;
    if (hwarp) warp_scan_incl2(inc, inch); else inc = warp_scan_incl(inc);
    if (lane == 31) { wtot[0][wid] = inc; wtot[1][wid] = inch; mbar_arrive(mbar); }      // 8 arrivals complete the phase

    // ---- exclusive prefix Q of the run totals: the tile's 256 runs, then the nh halo runs ----
    mbar_wait(mbar, parity);
    float below = 0.f, belowh = 0.f, total = 0.f;
    {
        const float4 a0 = *reinterpret_cast<const float4 *>(&wtot[0][0]), a1 = *reinterpret_cast<const float4 *>(&wtot[0][4]);
        const float w[8] = {a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w};
#pragma unroll
        for (int k = 0; k < 8; ++k) { if (k < wid) below += w[k]; total += w[k]; }
    }
    const float q_own = below + (inc - rt);                    // Q[tid]
    Q[tid] = q_own;
    if (hwarp) {
        const float4 a0 = *reinterpret_cast<const float4 *>(&wtot[1][0]), a1 = *reinterpret_cast<const float4 *>(&wtot[1][4]);
        const float w[8] = {a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w};
#pragma unroll
        for (int k = 0; k < 8; ++k) if (k < wid) belowh += w[k];
        if (tid <= nh) Q[ST_THREADS + tid] = total + belowh + (inch - ht);
    }
    mbar_arrive(mbar + 1);                                     // every thread wrote its Q entries: 256 arrivals

    // ---- the 16 windows that start at the thread's positions: sums of b and b^2.  de[k] = x[own + nmax + k] - x[own + k] is
    //      what a slide adds; it needs nothing from other warps, so it is formed before the wait for Q ----
    float de[ST_RUN - 1];
    if ((nmax & 3) == 0) {                                     // the entering samples as four 16-byte loads
        float e[ST_RUN];
        load16(xs, own + nmax, e);
#pragma unroll
        for (int k = 0; k < ST_RUN - 1; ++k) de[k] = e[k] - xo[k];
    } else {
#pragma unroll
        for (int k = 0; k < ST_RUN - 1; ++k) de[k] = xs[st_pad(own + nmax + k)] - xo[k];
    }
    float ps = 0.f;
    if (rem) {                                                 // the first rem values of run tid + q
        float p[ST_RUN];
        load16(xs, own + 16 * q, p);
#pragma unroll
        for (int k = 0; k < ST_RUN - 1; ++k) ps += (k < rem) ? p[k] - K : 0.f;
    }
    mbar_wait(mbar + 1, parity);
    if (FAST || wcnt > 0) {
        float b = (Q[tid + q] - q_own) + ps;
        float sb = b, sb2 = b * b;
#pragma unroll
        for (int k = 1; k < ST_RUN; ++k) {
            b += de[k - 1];
            if (FAST || k < wcnt) { sb += b; sb2 = fmaf(b, b, sb2); }
        }
        L.sb += (double)sb; L.sb2 += (double)sb2; L.nb += (double)wcnt;
    }
}

// dynamic shared memory of stats_partial_win: two landing buffers and the run-total prefix Q[2 * 256 + 1]
__host__ __device__ inline int st_win_xs_len(int nmax) { return st_pad(((ST_CHUNK + nmax - 1 + 3) & ~3) + ST_RUN); }
static size_t st_win_smem(int nmax) { return (size_t)(2 * st_win_xs_len(nmax) + 2 * ST_THREADS + 4) * sizeof(float); }

__global__ void __launch_bounds__(ST_THREADS, 3)
stats_partial_win(const float *__restrict__ x, int64_t n_dm, int64_t n_t, int64_t row_stride, int nmax,
                  Tri *__restrict__ part_x, Tri *__restrict__ part_b)
{
    x += (int64_t)blockIdx.y * row_stride;                     // per-row statistics: gridDim.y = rows (n_dm = 1 per slice)
    part_x += (size_t)blockIdx.y * gridDim.x;
    part_b += (size_t)blockIdx.y * gridDim.x;
    extern __shared__ __align__(16) unsigned char st_smem[];
    __shared__ Tri warp_acc[ST_THREADS / 32];
    __shared__ float red[2 * ST_THREADS / 32];
    __shared__ __align__(16) float wtot[2][ST_THREADS / 32];
    __shared__ unsigned long long mbar[2];                     // split barriers of a tile: warp totals written (8 arrivals), Q written (256)
    const int tid = threadIdx.x;
    if (tid == 0) {
        mbar_init(mbar, ST_THREADS / 32);
        mbar_init(mbar + 1, ST_THREADS);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    unsigned parity = 0;                                       // phase of both barriers: one phase per tile
    const int span = ST_CHUNK + nmax - 1;                      // samples staged per tile
    const int span4 = (span + 3) & ~3;
    const int xs_len = st_win_xs_len(nmax);
    float *xs0 = reinterpret_cast<float *>(st_smem);           // two landing buffers [st_pad(span4 + 16)]: raw samples, 0 past the row end
    float *Q = xs0 + 2 * xs_len;                               // [2 * 256 + 1] exclusive prefix of the run totals of x - K
    const int64_t nwin = n_t - nmax + 1;                       // full windows per row
    const int64_t tpr = (n_t + ST_CHUNK - 1) / ST_CHUNK;
    const int64_t total = n_dm * tpr;
    LaneAcc L;
    L.init();
    float K = 0.f;
    bool have_K = false;

    // (row, tile-in-row) of the persistent walk: the grid size is split once into whole rows and a remainder, so a step
    // is two adds and a wrap (a division per tile costs more instructions than a third of the tile's arithmetic)
    struct Pos { int64_t row; unsigned tr; };
    const unsigned utpr = (unsigned)tpr;
    const unsigned step_rows = gridDim.x / utpr, step_tiles = gridDim.x % utpr;
    auto advance = [&](Pos p) {
        p.tr += step_tiles; p.row += step_rows;
        if (p.tr >= utpr) { p.tr -= utpr; ++p.row; }
        return p;
    };
    // interior tile: whole tile + halo inside the row, and every row 16-byte aligned (else all tiles take the general path)
    const bool rows_aligned = ((reinterpret_cast<uintptr_t>(x) & 15) == 0) && ((row_stride & 3) == 0 || n_dm == 1);
    const unsigned tr_interior = (rows_aligned && n_t >= span4) ? (unsigned)((n_t - span4) / ST_CHUNK + 1) : 0u;   // tiles tr < this
    // stage a tile into landing buffer `buf` (asynchronous 16-byte copies; scalar loads at the row end / for unaligned rows).
    // Copy i of a thread moves floats [4 (tid + 256 i), + 4): 1024 floats further in global memory and, with one pad float4
    // per 16 floats, 1280 further in shared memory, so the loop is two pointer increments and the copy.
    const int n16 = span4 >> 2;
    const int dst_tid = st_pad(4 * tid);
    auto stage = [&](const Pos &p, int buf) {
        const int64_t t0 = (int64_t)p.tr * ST_CHUNK;
        const float *rp = x + p.row * row_stride;
        float *xb = xs0 + buf * xs_len;
        if (p.tr < tr_interior) {
            const float *src = rp + t0 + 4 * tid;
            float *dst = xb + dst_tid;
            for (int c = tid; c < n16; c += ST_THREADS, src += 4 * ST_THREADS, dst += 5 * ST_THREADS) cp_async16_st(dst, src);
        } else {
            const bool vec = ((reinterpret_cast<uintptr_t>(rp) & 15) == 0);
            for (int c = tid; c < n16; c += ST_THREADS) {
                const int64_t pos = t0 + 4 * c;
                float *dst = xb + st_pad(4 * c);
                if (vec && pos + 3 < n_t) cp_async16_st(dst, rp + pos);
                else {
#pragma unroll
                    for (int k = 0; k < 4; ++k) dst[k] = (pos + k < n_t) ? __ldg(rp + pos + k) : 0.0f;
                }
            }
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    int buf = 0;
    Pos pos = {(int64_t)(blockIdx.x / utpr), blockIdx.x % utpr};
    if ((int64_t)blockIdx.x < total) stage(pos, 0);

    for (int64_t c = blockIdx.x; c < total; c += gridDim.x, buf ^= 1) {
        const Pos cur = pos;
        const int64_t t0 = (int64_t)cur.tr * ST_CHUNK;
        pos = advance(pos);
        const float *xs = xs0 + buf * xs_len;
        asm volatile("cp.async.wait_group 0;" ::: "memory");
        __syncthreads();                                       // this tile has landed; everyone is done with the previous tile (other buffer, Q)
        if (c + gridDim.x < total) stage(pos, buf ^ 1);        // the next tile streams in while this one is reduced

        if (!have_K) {                                         // shift of this CTA: the mean of its first tile
            float xo[ST_RUN];
            load16(xs, ST_RUN * tid, xo);
            const int64_t left = n_t - (t0 + ST_RUN * tid);
            const int cnt = left >= ST_RUN ? ST_RUN : (left > 0 ? (int)left : 0);
            float s = 0.f;
            for (int k = 0; k < ST_RUN; ++k) if (k < cnt) s += xo[k];
            K = cta_mean(s, (float)cnt, red);
            have_K = true;
        }
        if (cur.tr < tr_interior) win_tile<true>(xs, Q, wtot, t0, n_t, nwin, nmax, K, L, mbar, parity);
        else win_tile<false>(xs, Q, wtot, t0, n_t, nwin, nmax, K, L, mbar, parity);
        parity ^= 1u;
    }
    L.flush();
    write_partial(warp_acc, L.acc, (double)K, 1.0, part_x + blockIdx.x, true);
    write_partial(warp_acc, L.windows(), (double)K, (double)nmax, part_b + blockIdx.x, true);
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
stats_finalize(const Tri *__restrict__ part_x, int count_x, const Tri *__restrict__ part_b, int count_b, int nmax_of_sigma,
               spd_stats_t *__restrict__ out)
{
    __shared__ Tri sh[ST_THREADS];
    Tri a = fold_partials(part_x, count_x, sh);
    Tri b = {0.0, 0.0, 0.0};
    if (count_b > 0) b = fold_partials(part_b, count_b, sh);
    if (threadIdx.x == 0) fill_stats(out, a, b, nmax_of_sigma);
}

// per-row variant of kernel 2: CTA r folds the partials of row r (a handful) in index order
__global__ void stats_finalize_rows(const Tri *__restrict__ part_x, const Tri *__restrict__ part_b, int per_row, int nmax_of_sigma,
                                    spd_stats_t *__restrict__ out)
{
    if (threadIdx.x != 0) return;
    const size_t r = blockIdx.x;
    Tri a = {0.0, 0.0, 0.0}, b = {0.0, 0.0, 0.0};
    for (int i = 0; i < per_row; ++i) {
        tri_merge(a, part_x[r * per_row + i]);
        if (nmax_of_sigma > 0) tri_merge(b, part_b[r * per_row + i]);
    }
    fill_stats(out + r, a, b, nmax_of_sigma);
}

// eq. 2 over whole results (the exchange step of a DM-row-sharded run), folded in index order.  Parts with no samples
// (a rank that holds no rows contributes an all-zero struct) are skipped, also in the nmax_of_sigma consistency check.
__global__ void stats_merge_kernel(const spd_stats_t *__restrict__ parts, int count, spd_stats_t *__restrict__ out)
{
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    Tri a = {0.0, 0.0, 0.0}, b = {0.0, 0.0, 0.0};
    int nm = -1;
    for (int i = 0; i < count; ++i) {
        if (parts[i].n == 0) continue;
        Tri pa = {(double)parts[i].n, parts[i].T, parts[i].S}, pb = {(double)parts[i].n_b, parts[i].T_b, parts[i].S_b};
        tri_merge(a, pa); tri_merge(b, pb);
        if (nm == -1) nm = parts[i].nmax_of_sigma;
        else if (parts[i].nmax_of_sigma != nm) nm = 0;
    }
    fill_stats(out, a, b, nm < 0 ? 0 : nm);
}

// stats_partial_win runs ONE resident wave of persistent CTAs.  Per device, the dynamic shared-memory limit is set once (to
// the largest tile, nmax = 4096) and the resident CTAs per SM of a shared-memory size are looked up once (the queries cost
// tens of microseconds per launch otherwise).
static cudaError_t stats_win_wave(size_t smem, int *wave)
{
    static std::mutex mu;
    static bool limit_set[64] = {};
    struct Entry { int dev; size_t smem; int wave; };
    static Entry cache[64];
    static int n_cached = 0;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    std::lock_guard<std::mutex> lk(mu);
    if (dev < 0 || dev >= 64 || !limit_set[dev]) {
        e = cudaFuncSetAttribute(stats_partial_win, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)st_win_smem(4096));
        if (e != cudaSuccess) return e;
        if (dev >= 0 && dev < 64) limit_set[dev] = true;
    }
    for (int i = 0; i < n_cached; ++i) if (cache[i].dev == dev && cache[i].smem == smem) { *wave = cache[i].wave; return cudaSuccess; }
    int sms = 0, per_sm = 0;
    if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
    if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, stats_partial_win, ST_THREADS, smem)) != cudaSuccess) return e;
    if (per_sm < 1) return cudaErrorInvalidConfiguration;
    *wave = sms * per_sm < MAX_PARTIALS ? sms * per_sm : MAX_PARTIALS;
    if (n_cached < 64) cache[n_cached++] = Entry{dev, smem, *wave};
    return cudaSuccess;
}

cudaError_t launch_stats(const float *x, int64_t n_dm, int64_t n_t, int64_t row_stride, int nmax_for_sigma,
                         spd_stats_t *d_stats, void *d_ws, cudaStream_t s)
{
    Tri *px = reinterpret_cast<Tri *>(d_ws), *pb = px + MAX_PARTIALS;
    int gx = 0, gb = 0;
    if (nmax_for_sigma > 0) {
        const int64_t tiles = n_dm * ((n_t + ST_CHUNK - 1) / ST_CHUNK);
        const size_t smem = st_win_smem(nmax_for_sigma);
        int wave = 0;
        cudaError_t e = stats_win_wave(smem, &wave);
        if (e != cudaSuccess) return e;
        gx = gb = (int)(tiles < wave ? tiles : wave);
        stats_partial_win<<<gx, ST_THREADS, smem, s>>>(x, n_dm, n_t, row_stride, nmax_for_sigma, px, pb);
    } else {
        int64_t rows = n_dm, cols = n_t, stride = row_stride;
        if (row_stride == n_t) { cols = n_dm * n_t; rows = 1; stride = cols; }     // contiguous: one long row
        const int64_t chunks = rows * ((cols + ST_CHUNK - 1) / ST_CHUNK);
        gx = (int)(chunks < ST_GRID ? chunks : ST_GRID);
        stats_partial<<<gx, ST_THREADS, 0, s>>>(x, rows, cols, stride, px);
    }
    stats_finalize<<<1, ST_THREADS, 0, s>>>(px, gx, pb, gb, nmax_for_sigma, d_stats);
    return cudaGetLastError();
}

// ---- one (mu, sigma, sigma_nmax) per DM row (reading A3's alternative) ----
constexpr int ST_ROW_CTAS = 8;                                  // CTAs that share one row
size_t stats_rows_ws_bytes(int64_t n_dm) { return (size_t)n_dm * ST_ROW_CTAS * 2 * sizeof(Tri); }

cudaError_t launch_stats_rows(const float *x, int64_t n_dm, int64_t n_t, int64_t row_stride, int nmax_for_sigma,
                              spd_stats_t *d_stats_rows, void *d_ws, cudaStream_t s)
{
    const int64_t cpr = (n_t + ST_CHUNK - 1) / ST_CHUNK;
    const int gx = (int)(cpr < ST_ROW_CTAS ? cpr : ST_ROW_CTAS);
    Tri *px = reinterpret_cast<Tri *>(d_ws), *pb = px + (size_t)n_dm * gx;
    cudaError_t e;
    size_t smem = 0;
    if (nmax_for_sigma > 0) {
        smem = st_win_smem(nmax_for_sigma);
        int wave = 0;
        if ((e = stats_win_wave(smem, &wave)) != cudaSuccess) return e;
    }
    for (int64_t r0 = 0; r0 < n_dm; r0 += 65535) {               // grid.y limit
        const unsigned ny = (unsigned)(n_dm - r0 < 65535 ? n_dm - r0 : 65535);
        const float *xr = x + r0 * row_stride;
        if (nmax_for_sigma > 0)
            stats_partial_win<<<dim3(gx, ny), ST_THREADS, smem, s>>>(xr, 1, n_t, row_stride, nmax_for_sigma, px + (size_t)r0 * gx, pb + (size_t)r0 * gx);
        else
            stats_partial<<<dim3(gx, ny), ST_THREADS, 0, s>>>(xr, 1, n_t, row_stride, px + (size_t)r0 * gx);
    }
    stats_finalize_rows<<<(unsigned)n_dm, 32, 0, s>>>(px, pb, gx, nmax_for_sigma, d_stats_rows);
    return cudaGetLastError();
}

// ---- spd_stats_rows_noalloc: the per-row statistics with the block partials in memory the library itself owns ----
// Some users of this library run where device memory cannot be requested at all: a search stage plugged into a
// telescope's real-time pipeline is handed its input and output buffers by the host framework, which has already
// carved the whole card into its own pools and forbids stages to allocate (an allocation would also stall every other
// stage: cudaMalloc waits for the device).  Such a caller has no way to produce the workspace spd_stats_rows asks for.
// For them the partials live in this file-scope array instead: 3 MiB that every GPU which loads libspd.so holds until
// the process exits, whether or not this entry point is ever called.
//
// In host code `noalloc_scratch` is only a handle for the symbol, never a device address (a kernel handed it would fault,
// or, on a GPU that can reach host memory, quietly work on the wrong bytes).  The address on the current device comes
// from cudaGetSymbolAddress, looked up once per device and remembered.
constexpr size_t NOALLOC_SCRATCH_BYTES = (size_t)SPD_NOALLOC_MAX_ROWS * ST_ROW_CTAS * 2 * sizeof(Tri);
static __device__ __align__(256) unsigned char noalloc_scratch[NOALLOC_SCRATCH_BYTES];

static cudaError_t noalloc_scratch_address(void **out)
{
    static std::mutex mu;
    static void *known[64] = {};
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    std::lock_guard<std::mutex> lk(mu);
    if (dev >= 0 && dev < 64 && known[dev]) { *out = known[dev]; return cudaSuccess; }
    void *p = nullptr;
    if ((e = cudaGetSymbolAddress(&p, noalloc_scratch)) != cudaSuccess) return e;
    if (!p) return cudaErrorInvalidSymbol;
    if (dev >= 0 && dev < 64) known[dev] = p;
    *out = p;
    return cudaSuccess;
}

// Same kernels, grid and partial layout as launch_stats_rows; only where the partials live differs.  Nothing in the
// array has to be cleared between calls: every CTA stores its partial before the finalize kernel of the same call reads
// it, and slots beyond this call's n_dm * gx are never read.
cudaError_t launch_stats_rows_noalloc(const float *x, int64_t n_dm, int64_t n_t, int64_t row_stride, int nmax_for_sigma,
                                      spd_stats_t *d_stats_rows, cudaStream_t s)
{
    if (stats_rows_ws_bytes(n_dm) > NOALLOC_SCRATCH_BYTES) return cudaErrorInvalidValue;   // the C ABI has already refused it
    void *scratch = nullptr;
    cudaError_t e = noalloc_scratch_address(&scratch);
    if (e != cudaSuccess) return e;
    return launch_stats_rows(x, n_dm, n_t, row_stride, nmax_for_sigma, d_stats_rows, scratch, s);
}

cudaError_t launch_stats_merge(const spd_stats_t *parts, int count, spd_stats_t *out, cudaStream_t s)
{
    stats_merge_kernel<<<1, 32, 0, s>>>(parts, count, out);
    return cudaGetLastError();
}

}  // namespace spd
