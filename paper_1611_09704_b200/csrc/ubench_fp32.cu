// ubench_fp32.cu -- issue rates of the fp32 instructions the sweep's width loop is made of, measured on the box.
//
// Why it exists: the sweep (Algorithm 1) has no contraction and is bound by fp32 instruction issue for
// Nmax > ~24.  SURVEY.md 8(d) takes 148 SMs x 128 lanes x sm_max_mhz as the peak and 2 FMA-pipe
// lane-ops per (sample, width) pair as the work; this program measures what one SM sub-partition (SMSP) really
// sustains for each instruction of the loop and for the loop's own instruction mix, so that the distance between the
// kernel and that peak can be split into "what the instruction set costs" and "what the kernel loses".
//
// Method: every thread keeps 16 independent accumulators (8 for packed ops) in registers and runs `iters` iterations
// of 4 unrolled repetitions of the body; one CTA = 128 threads = one warp per SMSP; the grid is 148 x k CTAs with
// k = 1, 2, 4, 8 resident CTAs per SM (dynamic shared memory pins the residency to exactly k).  Time is taken with
// CUDA events around the launch; the SM clock comes from clock64() against %globaltimer inside the same launch.
//   cycles per warp-instruction per SMSP = elapsed_ns * sm_ghz / (iters * 4 * instructions_per_repetition * k)
// `instructions_per_repetition` is what the SASS of the loop holds (check with cuobjdump -sass; the loop overhead of
// 3 instructions per 4 repetitions is not counted, which overstates the cost by < 2 %).
//
// Build / run:  python -m paper_1611_09704_b200.build --ubench && paper_1611_09704_b200/ubench_fp32
#include <cstdio>
#include <cstdlib>
#include <cuda_runtime.h>

#define CK(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) { fprintf(stderr, "%s: %s\n", #x, cudaGetErrorString(e_)); exit(1); } } while (0)

constexpr int NA = 16;          // independent scalar accumulators per thread
constexpr int REPS = 4;

__device__ __forceinline__ float fmax3(float a, float b, float c) { return fmaxf(fmaxf(a, b), c); }

enum Mode { FADD, FMUL, FFMA, FMNMX, FMNMX3, FADD2, FMUL2, FMUL2_BCAST, FFMA2, MIX_SCALAR, MIX_SCALAR_RCONST, MIX_PACKED, MIX_PACKED_RCONST, MIX_PACKED_RCONST_ARGMAX, LOP3_OP, IADD3_OP, MIX_NARROW, MIX_NARROW_TAGONLY, NMODES };
static const char *mode_name[NMODES] = {
    "FADD  r,r", "FMUL  r,r", "FFMA  r,r,r", "FMNMX r,r x2 (ptxas fuses two into one FMNMX3)", "FMNMX3 r,r,r", "FADD2 rr,rr", "FMUL2 rr,rr", "FMUL2 rr,r (scalar broadcast)",
    "FFMA2 rr,rr,rr", "loop mix, scalar: 2 FADD + 2 FMUL + 1 FMNMX3 per 2 pairs", "loop mix, scalar, r_w from the constant bank",
    "loop mix, packed: 2 FADD2 + 2 FMUL2(bcast) + 2 FMNMX3 per 4 pairs", "loop mix, packed, r_w from the constant bank (uniform register)",
    "loop mix, packed, r_w constant, + block arg-max (ping-pong maxima, FSETP + SEL per sum per 8 widths)",
    "LOP3 r,r,r", "IADD3 r,r",
    "narrow mix (sweep8_tagged): loop mix + per pair one LOP3 tag and half an FMNMX3 over the tagged values",
    "narrow mix without the exact maximum (tagged maximum only; not used: the SNR would lose its 5 low bits)"};
// warp instructions per repetition, and (sample, width) pairs per repetition per lane (0 = not a loop mix)
static const int mode_instr[NMODES] = {16, 16, 16, 8, 16, 8, 8, 8, 8, 40, 40, 48, 48, 112, 16, 16, 96, 80};
static const int mode_pairs[NMODES] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 16, 16, 32, 32, 64, 0, 0, 32, 32};

struct RTable { float r[8]; };

template <int MODE>
__global__ void __launch_bounds__(128) bench_kernel(float *out, long long *clk, int iters, float fa, float fb, RTable rt, int tagmask)
{
    extern __shared__ float dummy[];
    float a[NA], w[NA], m[NA];
#pragma unroll
    for (int j = 0; j < NA; ++j) { a[j] = fa * (threadIdx.x + j); w[j] = fb * (j + 1) + threadIdx.x * 1e-3f; m[j] = -1e30f + threadIdx.x + j; }
    float2 A2[8], W2[8], M2[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) { A2[j] = make_float2(a[j], a[j + 8]); W2[j] = make_float2(w[j], w[j + 8]); M2[j] = make_float2(m[j], m[j + 8]); }
    const float r0 = rt.r[0] * fb, r1 = rt.r[1] * fb;      // in registers
    float2 O2[8]; int wx[8], wy[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) { O2[j] = M2[j]; wx[j] = 0; wy[j] = 0; }
    long long t0 = 0, g0 = 0;
    if (threadIdx.x == 0) { asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g0)); t0 = clock64(); }
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int rep = 0; rep < (MODE == MIX_PACKED_RCONST_ARGMAX ? 0 : REPS); ++rep) {
            if (MODE == FADD) {
#pragma unroll
                for (int j = 0; j < NA; ++j) a[j] = __fadd_rn(a[j], w[j]);
            } else if (MODE == FMUL) {
#pragma unroll
                for (int j = 0; j < NA; ++j) a[j] = __fmul_rn(a[j], w[j]);
            } else if (MODE == FFMA) {
#pragma unroll
                for (int j = 0; j < NA; ++j) a[j] = __fmaf_rn(a[j], w[j], m[j]);
            } else if (MODE == FMNMX) {
#pragma unroll
                for (int j = 0; j < NA; ++j) a[j] = fmaxf(a[j], w[(j + 5 * rep) & 15]);
            } else if (MODE == FMNMX3) {
#pragma unroll
                for (int j = 0; j < NA; ++j) a[j] = fmax3(a[j], w[j], m[j]);
            } else if (MODE == FADD2) {
#pragma unroll
                for (int j = 0; j < 8; ++j) A2[j] = __fadd2_rn(A2[j], W2[j]);
            } else if (MODE == FMUL2) {
#pragma unroll
                for (int j = 0; j < 8; ++j) A2[j] = __fmul2_rn(A2[j], W2[j]);
            } else if (MODE == FMUL2_BCAST) {
#pragma unroll
                for (int j = 0; j < 8; ++j) A2[j] = __fmul2_rn(A2[j], make_float2(r0, r0));
            } else if (MODE == FFMA2) {
#pragma unroll
                for (int j = 0; j < 8; ++j) A2[j] = __ffma2_rn(A2[j], W2[j], M2[j]);
            } else if (MODE == MIX_SCALAR || MODE == MIX_SCALAR_RCONST) {
                // the width loop of the sweep for 8 running sums and 2 widths, scalar form (w[] plays the sliding window)
                const float q0 = (MODE == MIX_SCALAR_RCONST) ? rt.r[2 * rep] : r0, q1 = (MODE == MIX_SCALAR_RCONST) ? rt.r[2 * rep + 1] : r1;
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    a[j] = __fadd_rn(a[j], w[(j + 2 * rep) & 15]);
                    const float s0 = __fmul_rn(a[j], q0);
                    a[j] = __fadd_rn(a[j], w[(j + 2 * rep + 1) & 15]);
                    const float s1 = __fmul_rn(a[j], q1);
                    m[j] = fmax3(m[j], s0, s1);
                }
            } else if (MODE == LOP3_OP) {
#pragma unroll
                for (int j = 0; j < NA; ++j) { int d; asm volatile("lop3.b32 %0, %1, %2, %3, 0xEA;" : "=r"(d) : "r"(__float_as_int(a[j])), "r"(__float_as_int(w[j])), "r"(__float_as_int(m[j]))); a[j] = __int_as_float(d); }
            } else if (MODE == IADD3_OP) {
#pragma unroll
                for (int j = 0; j < NA; ++j) { int d; asm volatile("add.s32 %0, %1, %2;" : "=r"(d) : "r"(__float_as_int(a[j])), "r"(__float_as_int(w[j]))); a[j] = __int_as_float(d); }
            } else if (MODE == MIX_NARROW || MODE == MIX_NARROW_TAGONLY) {
                // the width loop of boxcar_snr_sweep_narrow: the loop mix plus a second maximum over values whose 5 low mantissa
                // bits carry the width (one LOP3 per value); O2 plays the tagged maxima
                const float2 q0 = make_float2(rt.r[2 * rep], rt.r[2 * rep]), q1 = make_float2(rt.r[2 * rep + 1], rt.r[2 * rep + 1]);
                const int c0 = 31 - 2 * rep, c1 = c0 - 1;
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    A2[j] = __fadd2_rn(A2[j], W2[(j + 2 * rep) & 7]);
                    const float2 s0 = __fmul2_rn(A2[j], q0);
                    A2[j] = __fadd2_rn(A2[j], W2[(j + 2 * rep + 1) & 7]);
                    const float2 s1 = __fmul2_rn(A2[j], q1);
                    if (MODE == MIX_NARROW) { M2[j].x = fmax3(M2[j].x, s0.x, s1.x); M2[j].y = fmax3(M2[j].y, s0.y, s1.y); }
                    float t0, t1, t2, t3;
                    asm("lop3.b32 %0, %1, %2, %3, 0xEA;" : "=f"(t0) : "f"(s0.x), "r"(tagmask), "r"(c0));
                    asm("lop3.b32 %0, %1, %2, %3, 0xEA;" : "=f"(t1) : "f"(s1.x), "r"(tagmask), "r"(c1));
                    asm("lop3.b32 %0, %1, %2, %3, 0xEA;" : "=f"(t2) : "f"(s0.y), "r"(tagmask), "r"(c0));
                    asm("lop3.b32 %0, %1, %2, %3, 0xEA;" : "=f"(t3) : "f"(s1.y), "r"(tagmask), "r"(c1));
                    O2[j].x = fmax3(O2[j].x, t0, t1); O2[j].y = fmax3(O2[j].y, t2, t3);
                }
            } else if (MODE == MIX_PACKED || MODE == MIX_PACKED_RCONST) {
                // the same for 8 packed running sums (two samples each): what sweep8 in sweep.cu issues
                const bool rc = (MODE != MIX_PACKED);
                const float2 q0 = rc ? make_float2(rt.r[2 * rep], rt.r[2 * rep]) : make_float2(r0, r0);
                const float2 q1 = rc ? make_float2(rt.r[2 * rep + 1], rt.r[2 * rep + 1]) : make_float2(r1, r1);
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    A2[j] = __fadd2_rn(A2[j], W2[(j + 2 * rep) & 7]);
                    const float2 s0 = __fmul2_rn(A2[j], q0);
                    A2[j] = __fadd2_rn(A2[j], W2[(j + 2 * rep + 1) & 7]);
                    const float2 s1 = __fmul2_rn(A2[j], q1);
                    M2[j].x = fmax3(M2[j].x, s0.x, s1.x); M2[j].y = fmax3(M2[j].y, s0.y, s1.y);
                }
            }
        }
        if (MODE == MIX_PACKED_RCONST_ARGMAX) {
            // two blocks of 8 widths as in boxcar_snr_sweep: the running maximum ping-pongs between M2 and O2 so that the
            // values before and after a block are both live; FSETP + SEL per running sum record the block that raised it
#pragma unroll
            for (int half = 0; half < 2; ++half) {
                float2 (&in)[8] = half ? O2 : M2;
                float2 (&ot)[8] = half ? M2 : O2;
#pragma unroll
                for (int rep = 0; rep < REPS; ++rep) {
                    const float2 q0 = make_float2(rt.r[2 * rep], rt.r[2 * rep]), q1 = make_float2(rt.r[2 * rep + 1], rt.r[2 * rep + 1]);
#pragma unroll
                    for (int j = 0; j < 8; ++j) {
                        A2[j] = __fadd2_rn(A2[j], W2[(j + 2 * rep) & 7]);
                        const float2 s0 = __fmul2_rn(A2[j], q0);
                        A2[j] = __fadd2_rn(A2[j], W2[(j + 2 * rep + 1) & 7]);
                        const float2 s1 = __fmul2_rn(A2[j], q1);
                        const float2 mm = rep == 0 ? in[j] : ot[j];
                        ot[j].x = fmax3(mm.x, s0.x, s1.x); ot[j].y = fmax3(mm.y, s0.y, s1.y);
                    }
                }
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    wx[j] = (ot[j].x > in[j].x) ? 2 * it + half : wx[j];
                    wy[j] = (ot[j].y > in[j].y) ? 2 * it + half : wy[j];
                }
            }
        }
    }
    if (threadIdx.x == 0) {
        long long t1 = clock64(), g1;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g1));
        if (blockIdx.x == 0) { clk[0] = t1 - t0; clk[1] = g1 - g0; }
    }
    float acc = 0.f;
#pragma unroll
    for (int j = 0; j < NA; ++j) acc += a[j] + m[j] + w[j];
#pragma unroll
    for (int j = 0; j < 8; ++j) acc += A2[j].x + A2[j].y + M2[j].x + M2[j].y + O2[j].x + O2[j].y + (float)(wx[j] + wy[j]);
    if (acc == 1.2345f) out[threadIdx.x] = acc + dummy[0];
}

template <int MODE>
static void run_mode(int k, float *d_out, long long *d_clk, int sms, int smem_per_sm)
{
    const int smem = smem_per_sm / k - 2048;                       // exactly k CTAs fit on an SM
    CK(cudaFuncSetAttribute(bench_kernel<MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    int occ = 0;
    CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, bench_kernel<MODE>, 128, smem));
    RTable rt;
    for (int i = 0; i < 8; ++i) rt.r[i] = 1.0f / (1.0f + 0.001f * i);
    const int iters = 1 << 15;
    cudaEvent_t e0, e1;
    CK(cudaEventCreate(&e0)); CK(cudaEventCreate(&e1));
    float best_ms = 1e30f; long long clk[2] = {0, 0};
    for (int t = 0; t < 4; ++t) {                                  // first run is the warm-up; best of the next three
        CK(cudaEventRecord(e0));
        bench_kernel<MODE><<<sms * k, 128, smem>>>(d_out, d_clk, iters, 1.0f, 1.000001f, rt, ~31);
        CK(cudaEventRecord(e1));
        CK(cudaEventSynchronize(e1));
        float ms; CK(cudaEventElapsedTime(&ms, e0, e1));
        if (t > 0 && ms < best_ms) { best_ms = ms; CK(cudaMemcpy(clk, d_clk, sizeof clk, cudaMemcpyDeviceToHost)); }
    }
    const double ghz = (double)clk[0] / (double)clk[1];
    const double cyc = best_ms * 1e6 * ghz;                        // SM cycles of the launch
    const double per_instr = cyc / ((double)iters * REPS * mode_instr[MODE] * k);
    printf("%-66s | %d | %4d | %7.3f | %8.3f |", mode_name[MODE], k, occ, best_ms, ghz * 1e3);
    printf(" %6.3f |", per_instr);
    if (mode_pairs[MODE]) printf(" %6.3f |", cyc / ((double)iters * REPS * mode_pairs[MODE] * k)); else printf("      - |");
    printf("\n");
    CK(cudaEventDestroy(e0)); CK(cudaEventDestroy(e1));
}

template <int MODE>
static void run_all(float *d_out, long long *d_clk, int sms, int smem_per_sm)
{
    for (int k : {1, 2, 4, 8}) run_mode<MODE>(k, d_out, d_clk, sms, smem_per_sm);
}

int main()
{
    cudaDeviceProp p; CK(cudaGetDeviceProperties(&p, 0));
    float *d_out; long long *d_clk;
    CK(cudaMalloc(&d_out, 4096)); CK(cudaMalloc(&d_clk, 64));
    const int sms = p.multiProcessorCount, smem_per_sm = (int)p.sharedMemPerMultiprocessor;
    printf("device: %s, %d SMs, clockRate %d kHz\n", p.name, sms, p.clockRate);
    printf("one CTA = 128 threads = 1 warp per SMSP; k = resident CTAs per SM = warps per SMSP\n");
    printf("%-66s | k | occ | ms      | SM MHz   | clk/warp-instr/SMSP | clk per 32 pairs |\n", "body");
    run_all<FADD>(d_out, d_clk, sms, smem_per_sm);
    run_all<FMUL>(d_out, d_clk, sms, smem_per_sm);
    run_all<FFMA>(d_out, d_clk, sms, smem_per_sm);
    run_all<FMNMX>(d_out, d_clk, sms, smem_per_sm);
    run_all<FMNMX3>(d_out, d_clk, sms, smem_per_sm);
    run_all<FADD2>(d_out, d_clk, sms, smem_per_sm);
    run_all<FMUL2>(d_out, d_clk, sms, smem_per_sm);
    run_all<FMUL2_BCAST>(d_out, d_clk, sms, smem_per_sm);
    run_all<FFMA2>(d_out, d_clk, sms, smem_per_sm);
    run_all<MIX_SCALAR>(d_out, d_clk, sms, smem_per_sm);
    run_all<MIX_SCALAR_RCONST>(d_out, d_clk, sms, smem_per_sm);
    run_all<MIX_PACKED>(d_out, d_clk, sms, smem_per_sm);
    run_all<MIX_PACKED_RCONST>(d_out, d_clk, sms, smem_per_sm);
    run_all<MIX_PACKED_RCONST_ARGMAX>(d_out, d_clk, sms, smem_per_sm);
    run_all<LOP3_OP>(d_out, d_clk, sms, smem_per_sm);
    run_all<IADD3_OP>(d_out, d_clk, sms, smem_per_sm);
    run_all<MIX_NARROW>(d_out, d_clk, sms, smem_per_sm);
    run_all<MIX_NARROW_TAGONLY>(d_out, d_clk, sms, smem_per_sm);
    return 0;
}
