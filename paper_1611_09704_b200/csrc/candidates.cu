// candidates.cu -- step 4b: candidate selection (section 2.4; readings A12-A15).
//
// Every (d, t) of the max-over-width SNR plane with snr >= f_T becomes one 16-byte record (dm, t, snr, width);
// the planes are not modified and the list is unordered.  Pure HBM stream: 4 B/sample read; the width plane is
// touched only at hits.  Hits are rare, so the fast path is loads + compares + one warp vote; records are
// appended with one atomicAdd per warp that has any hit (warp-aggregated), written as one 128-bit store.
#include "spd_common.cuh"

namespace spd {

constexpr int CD_THREADS = 256;
constexpr int CD_VEC     = 4;                         // float4 loads in flight per thread
constexpr int CD_CHUNK   = CD_THREADS * CD_VEC * 4;   // 4096 samples per CTA iteration
constexpr int CD_GRID    = 148 * 8;

__device__ __forceinline__ float4 ldg_stream4c(const float *p)
{
    float4 v;
    asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];"
                 : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
    return v;
}

__global__ void zero_count_kernel(unsigned long long *count) { *count = 0ULL; }

__global__ void __launch_bounds__(CD_THREADS)
candidates_compact(const float *__restrict__ snr, const uint16_t *__restrict__ width, int64_t n_dm, int64_t n_t,
                   int64_t row_stride, float thr, spd_candidate_t *__restrict__ out, unsigned long long capacity,
                   unsigned long long *__restrict__ count, uint32_t t_scale /* record.t = t_scale * sample index (decimated levels) */)
{
    const int tid = threadIdx.x;
    const int64_t cpr = (n_t + CD_CHUNK - 1) / CD_CHUNK;
    const int64_t total = n_dm * cpr;
    for (int64_t c = blockIdx.x; c < total; c += gridDim.x) {
        const int64_t row = c / cpr, off = (c - row * cpr) * CD_CHUNK;
        const float *base = snr + row * row_stride;
        const bool full = (off + CD_CHUNK <= n_t) && ((reinterpret_cast<uintptr_t>(base + off) & 15) == 0);
        float v[CD_VEC][4];
        if (full) {
#pragma unroll
            for (int k = 0; k < CD_VEC; ++k) {
                float4 q = ldg_stream4c(base + off + (k * CD_THREADS + tid) * 4);
                v[k][0] = q.x; v[k][1] = q.y; v[k][2] = q.z; v[k][3] = q.w;
            }
        } else {
#pragma unroll
            for (int k = 0; k < CD_VEC; ++k)
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    int64_t p = off + (int64_t)(k * CD_THREADS + tid) * 4 + e;
                    v[k][e] = (p < n_t) ? __ldg(base + p) : __int_as_float(0xff800000);
                }
        }
        bool any = false;
#pragma unroll
        for (int k = 0; k < CD_VEC; ++k)
#pragma unroll
            for (int e = 0; e < 4; ++e) any |= (v[k][e] >= thr);
        if (__any_sync(0xffffffffu, any)) {
#pragma unroll
            for (int k = 0; k < CD_VEC; ++k)
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const int64_t p = off + (int64_t)(k * CD_THREADS + tid) * 4 + e;
                    const bool hit = v[k][e] >= thr;
                    uint32_t w = 0;
                    if (hit && width) w = width[row * row_stride + p];
                    append_candidate(hit, (uint32_t)row, (uint32_t)p * t_scale, v[k][e], w, out, capacity, count);
                }
        }
    }
}

cudaError_t launch_candidates(const float *snr, const uint16_t *width, int64_t n_dm, int64_t n_t, int64_t row_stride,
                              float threshold, spd_candidate_t *out, unsigned long long capacity,
                              unsigned long long *d_count, cudaStream_t s, bool zero_count, uint32_t t_scale)
{
    if (zero_count) zero_count_kernel<<<1, 1, 0, s>>>(d_count);
    int64_t rows = n_dm, cols = n_t, stride = row_stride;
    const int64_t chunks = rows * ((cols + CD_CHUNK - 1) / CD_CHUNK);
    const int g = (int)(chunks < CD_GRID ? chunks : CD_GRID);
    if (chunks <= 0) return cudaGetLastError();
    candidates_compact<<<g, CD_THREADS, 0, s>>>(snr, width, rows, cols, stride, threshold, out, capacity, d_count, t_scale);
    return cudaGetLastError();
}

}  // namespace spd
