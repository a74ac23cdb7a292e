// lpm_probe.cu — micro-benchmarks behind lpm_probe(): the MEASURED denominators of the rooflines
// bench.py reports ("replace 3.72e13 by a measured FP32-FMA and mul.wide.u32 issue
// rate"; "the three micro-benchmarks [conflict-free shared atomicAdd, random-address red.global.add
// over the same footprint, same-address service time] are part of the deliverable").  Each probe
// runs a few warm-up launches, then times `reps` launches with CUDA events on the given stream and
// returns operations per second.  No probe touches a simulation handle.
#include "lpm_internal.h"

namespace lpm {

namespace {

constexpr int kThreads = 256;

// 0: dependent-chain-free FFMA stream, 8 independent accumulators per thread
__global__ void __launch_bounds__(kThreads) probe_ffma(float *out, int iters, float a, float b)
{
    float r[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) r[i] = (float)(threadIdx.x + i);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 4; ++u)
#pragma unroll
            for (int i = 0; i < 8; ++i) r[i] = fmaf(r[i], a, b);
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += r[i];
    if (s == 123.456f) out[0] = s;
}

// 1: the Philox round mix: one IMAD.WIDE.U32 + one LOP3 per op pair, 4 independent chains
__global__ void __launch_bounds__(kThreads) probe_imad(uint32_t *out, int iters, uint32_t k)
{
    uint32_t c[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) c[i] = threadIdx.x * 4 + i;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u)
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const uint64_t p = (uint64_t)0xD2511F53u * c[i];
                c[i] = (uint32_t)(p >> 32) ^ (uint32_t)p ^ k;
            }
    }
    if ((c[0] ^ c[1] ^ c[2] ^ c[3]) == 0x12345678u) out[0] = c[0];
}

__device__ __forceinline__ uint32_t lcg(uint32_t &s) { s = s * 1664525u + 1013904223u; return s; }

// 2: random-address red.global.add.f64 over `cells` doubles (deposit map / concentration sums)
__global__ void __launch_bounds__(kThreads) probe_red_f64(double *buf, uint64_t cells, int iters)
{
    uint32_t s = (blockIdx.x * kThreads + threadIdx.x) * 2654435761u + 12345u;
    for (int it = 0; it < iters; ++it) {
        const uint64_t i = ((uint64_t)lcg(s) * cells) >> 32;
        atomicAdd(buf + i, 1.0);
    }
}

// 3: random-address red.global.add.u32 over `cells` words (particle counts)
__global__ void __launch_bounds__(kThreads) probe_red_u32(uint32_t *buf, uint64_t cells, int iters)
{
    uint32_t s = (blockIdx.x * kThreads + threadIdx.x) * 2654435761u + 777u;
    for (int it = 0; it < iters; ++it) {
        const uint64_t i = ((uint64_t)lcg(s) * cells) >> 32;
        atomicAdd(buf + i, 1u);
    }
}

// 4: every thread of the grid adds to ONE address (hottest-cell service time)
__global__ void __launch_bounds__(kThreads) probe_red_same(double *buf, int iters)
{
    for (int it = 0; it < iters; ++it) atomicAdd(buf, 1.0);
}

// 5: conflict-free shared atomicAdd (u32, native ATOMS.ADD): lane i hits bank i
__global__ void __launch_bounds__(kThreads) probe_atoms(uint32_t *out, int iters)
{
    __shared__ uint32_t sm[kThreads];
    sm[threadIdx.x] = 0;
    __syncthreads();
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u) atomicAdd(&sm[(threadIdx.x + 32 * u) & (kThreads - 1)], 1u);
    }
    __syncthreads();
    if (sm[threadIdx.x] == 0xffffffffu) out[0] = 1;
}

// 6: 16-byte gathers, every lane its own 32-byte sector inside an L1-resident window (the met gather
// of a warp whose lanes sit in different cells): L1 data-pipe sectors per second
__global__ void __launch_bounds__(kThreads) probe_gather(const float4 *buf, uint32_t texels, float *out, int iters)
{
    uint32_t s = (blockIdx.x * kThreads + threadIdx.x) * 2654435761u + 99u;
    float acc = 0.f;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            const uint32_t i = (lcg(s) >> 8) % texels;
            const float4 v = __ldg(buf + i);
            acc += v.x + v.w;
        }
    }
    if (acc == 123.456f) out[0] = acc;
}

// 7: the alternative to the L1 gathers that north_star names ("staged ... into shared memory"): 16-byte LDS gathers, every lane its own
// texel inside a window of `texels` float4 in shared memory (a warp's block of columns x levels, staged per step): LDS.128 lane-loads
// per second.  One trilinear sample needs 8 of them (or 4 of 32 bytes from global memory, probe 6 with 32-byte texels).
__global__ void __launch_bounds__(kThreads) probe_smem_gather(float *out, uint32_t texels, int iters)
{
    __shared__ float4 win[1024];
    for (int i = threadIdx.x; i < 1024; i += kThreads) win[i] = make_float4((float)i, 1.f, 2.f, 3.f);
    __syncthreads();
    uint32_t s = (blockIdx.x * kThreads + threadIdx.x) * 2654435761u + 4242u;
    float acc = 0.f;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            const uint32_t i = (lcg(s) >> 8) % texels;
            const float4 v = win[i];
            acc += v.x + v.w;
        }
    }
    if (acc == 123.456f) out[0] = acc;
}

// 8: 32-byte gathers (ld.global.nc.v8.f32), every lane its own sector of an L1-resident window: the z-pair texel gather of the step kernel
__global__ void __launch_bounds__(kThreads) probe_gather32(const float4 *buf, uint32_t texels, float *out, int iters)
{
    uint32_t s = (blockIdx.x * kThreads + threadIdx.x) * 2654435761u + 77u;
    float acc = 0.f;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const uint32_t i = (lcg(s) >> 8) % texels;
            float a0, a1, a2, a3, a4, a5, a6, a7;
            asm volatile("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                         : "=f"(a0), "=f"(a1), "=f"(a2), "=f"(a3), "=f"(a4), "=f"(a5), "=f"(a6), "=f"(a7) : "l"(buf + 2ull * i));
            acc += (a0 + a1) + (a2 + a3) + (a4 + a5) + (a6 + a7);
        }
    }
    if (acc == 123.456f) out[0] = acc;
}

}  // namespace

// returns operations per second in *ops (FMA lane-ops, IMAD+LOP3 lane-op pairs x2, atomics, sectors)
cudaError_t run_probe(int kind, uint64_t footprint_bytes, void *scratch_dev, uint64_t scratch_bytes, int reps, double *ops,
                      cudaStream_t st)
{
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int blocks = sms * 8;
    const uint64_t threads = (uint64_t)blocks * kThreads;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    if (footprint_bytes > scratch_bytes) footprint_bytes = scratch_bytes;
    double per_launch = 0.0;
    cudaError_t rc = cudaSuccess;
    for (int pass = 0; pass < 2 && rc == cudaSuccess; ++pass) {  // pass 0 = warm-up
        const int n = pass == 0 ? 2 : reps;
        if (pass == 1) cudaEventRecord(e0, st);
        for (int r = 0; r < n; ++r) {
            switch (kind) {
                case 0: probe_ffma<<<blocks, kThreads, 0, st>>>((float *)scratch_dev, 2048, 1.0000001f, 1e-7f); per_launch = (double)threads * 2048 * 32; break;
                case 1: probe_imad<<<blocks, kThreads, 0, st>>>((uint32_t *)scratch_dev, 1024, 0x9E3779B9u); per_launch = (double)threads * 1024 * 32 * 2; break;
                case 2: probe_red_f64<<<blocks, kThreads, 0, st>>>((double *)scratch_dev, footprint_bytes / 8, 256); per_launch = (double)threads * 256; break;
                case 3: probe_red_u32<<<blocks, kThreads, 0, st>>>((uint32_t *)scratch_dev, footprint_bytes / 4, 256); per_launch = (double)threads * 256; break;
                case 4: probe_red_same<<<blocks, kThreads, 0, st>>>((double *)scratch_dev, 16); per_launch = (double)threads * 16; break;
                case 5: probe_atoms<<<blocks, kThreads, 0, st>>>((uint32_t *)scratch_dev, 512); per_launch = (double)threads * 512 * 8; break;
                case 6: probe_gather<<<blocks, kThreads, 0, st>>>((const float4 *)scratch_dev, (uint32_t)(footprint_bytes / 16), (float *)scratch_dev + scratch_bytes / 4 - 4, 128); per_launch = (double)threads * 128 * 8; break;
                case 7: probe_smem_gather<<<blocks, kThreads, 0, st>>>((float *)scratch_dev, (uint32_t)(footprint_bytes / 16 < 1024 ? (footprint_bytes / 16 ? footprint_bytes / 16 : 1) : 1024), 256); per_launch = (double)threads * 256 * 8; break;
                case 8: probe_gather32<<<blocks, kThreads, 0, st>>>((const float4 *)scratch_dev, (uint32_t)(footprint_bytes / 32), (float *)scratch_dev + scratch_bytes / 4 - 4, 128); per_launch = (double)threads * 128 * 4; break;
                default: rc = cudaErrorInvalidValue; break;
            }
            if (rc != cudaSuccess) break;
        }
        if (rc == cudaSuccess) rc = cudaGetLastError();
    }
    cudaEventRecord(e1, st);
    if (rc == cudaSuccess) rc = cudaEventSynchronize(e1);
    float ms = 0.f;
    if (rc == cudaSuccess) rc = cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (rc == cudaSuccess) *ops = ms > 0.f ? per_launch * reps / ((double)ms * 1e-3) : 0.0;
    return rc;
}

}  // namespace lpm
