// lpm_bin.cu — concentration binning, read-out and utility kernels.
//
// P:L108 "Activities or masses of particles are summarized on a rectangular grid"; the paper does
// this on the CPU after a D2H copy and suggests a separate GPU kernel.  Here the
// particles never leave HBM.  Cell rule R10 (exact fp32 index), counts in u32 (exact), sums of the
// stored q in fp64 so that the result does not depend on the order of the atomics beyond 1e-16.
#include <curand_kernel.h>

#include "lpm_device.cuh"

namespace lpm {

// v0: one particle per thread iteration, warp-aggregated: lanes that hit the same cell are
// combined with match.any so that the hot cells next to the source cost one RED per warp.
__global__ void __launch_bounds__(256) bin_kernel(const __grid_constant__ BinArgs A)
{
    const uint64_t n = A.n_dev ? *A.n_dev : A.n;
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    const uint64_t n_round = (n + 31) & ~(uint64_t)31;  // keep warps converged for match.any
    const int lane = threadIdx.x & 31;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_round; i += stride) {
        int cell = -1;
        float q0 = 0.f, q1 = 0.f;
        if (i < n) {
            const float4 p = A.xyzq[i];
            if (p.z >= 0.0f) {  // z < 0 marks an exited slot
                const int ci = cell_of(p.x, A.cg.x0, A.cg.inv_dx, A.cg.nx);
                const int cj = cell_of(p.y, A.cg.y0, A.cg.inv_dy, A.cg.ny);
                const int ck = cell_of(p.z, A.cg.z0, A.cg.inv_dz, A.cg.nz);
                if ((ci | cj | ck) >= 0) {
                    cell = (ck * A.cg.ny + cj) * A.cg.nx + ci;
                    q0 = p.w;
                    if (A.K > 1) q1 = A.q1[i];
                }
            }
        }
        const uint32_t peers = __match_any_sync(0xffffffffu, cell);
        if (cell < 0) continue;
        const int leader = __ffs(peers) - 1;
        // sum q over the peer group in lane order (deterministic for a given warp content)
        double s0 = 0.0, s1 = 0.0;
        uint32_t rest = peers;
        while (rest) {
            const int src = __ffs(rest) - 1;
            rest &= rest - 1;
            s0 += (double)__shfl_sync(peers, q0, src);
            if (A.K > 1) s1 += (double)__shfl_sync(peers, q1, src);
        }
        if (lane == leader) {
            atomicAdd(A.cnt + cell, (uint32_t)__popc(peers));
            atomicAdd(A.conc + cell, s0);
            if (A.K > 1) atomicAdd(A.conc + A.cells3 + cell, s1);
        }
    }
}

cudaError_t launch_bin(const BinArgs &a, int blocks, cudaStream_t st)
{
    bin_kernel<<<blocks, 256, 0, st>>>(a);
    return cudaGetLastError();
}

// concentration read-out: Bq m^-3 = sum(q) * G_k(t_bin) / V   (scale[k] = G_k / V)
__global__ void conc_readout_kernel(const double *__restrict__ conc, float *__restrict__ out, uint64_t cells3,
                                    int K, double s0, double s1)
{
    const uint64_t total = cells3 * (uint64_t)K;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (uint64_t)gridDim.x * blockDim.x)
        out[i] = (float)(conc[i] * (i < cells3 ? s0 : s1));
}

cudaError_t launch_conc_readout(const double *conc, float *out, uint64_t cells3, int K, const double *scale, cudaStream_t st)
{
    const uint64_t total = cells3 * K;
    int blocks = (int)((total + 255) / 256 < 148 * 8 ? (total + 255) / 256 : 148 * 8);
    conc_readout_kernel<<<blocks < 1 ? 1 : blocks, 256, 0, st>>>(conc, out, cells3, K, scale[0], K > 1 ? scale[1] : 0.0);
    return cudaGetLastError();
}

// S 8(f)3 dose grid: dose[k][cell] += sum_q[k][cell] * G_k(t_b) / V * T_bin at every cadence binning
__global__ void dose_accum_kernel(const double *__restrict__ conc, double *__restrict__ dose, uint64_t cells3, int K, double s0, double s1)
{
    const uint64_t total = cells3 * (uint64_t)K;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (uint64_t)gridDim.x * blockDim.x) {
        const double c = conc[i];
        if (c != 0.0) dose[i] += c * (i < cells3 ? s0 : s1);
    }
}

cudaError_t launch_dose_accum(const double *conc, double *dose, uint64_t cells3, int K, const double *scale, cudaStream_t st)
{
    const uint64_t total = cells3 * K;
    int blocks = (int)((total + 255) / 256 < 148 * 8 ? (total + 255) / 256 : 148 * 8);
    dose_accum_kernel<<<blocks < 1 ? 1 : blocks, 256, 0, st>>>(conc, dose, cells3, K, scale[0], K > 1 ? scale[1] : 0.0);
    return cudaGetLastError();
}

__global__ void dep_readout_kernel(const double *__restrict__ dep, float *out32, double *out64, uint64_t cells2, uint64_t total, double s0, double s1)
{
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (uint64_t)gridDim.x * blockDim.x) {
        const double v = dep[i] * (i < cells2 ? s0 : s1);
        if (out32) out32[i] = (float)v;
        if (out64) out64[i] = v;
    }
}

// scale[k] = 1 / cell area, times the ground-decay factor of nuclide k since the map's reference time (R13)
cudaError_t launch_dep_readout(const double *dep, float *out_f32, double *out_f64, uint64_t cells2, int K, const double *scale, cudaStream_t st)
{
    const uint64_t total = cells2 * K;
    int blocks = (int)((total + 255) / 256 < 148 * 8 ? (total + 255) / 256 : 148 * 8);
    dep_readout_kernel<<<blocks < 1 ? 1 : blocks, 256, 0, st>>>(dep, out_f32, out_f64, cells2, total, scale[0], K > 1 ? scale[1] : 0.0);
    return cudaGetLastError();
}

// R13: move the reference time of one nuclide's ground-decaying map (keeps the stored values of the order of the activities)
__global__ void dep_rebase_kernel(double *dep, uint64_t cells2, double factor)
{
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < cells2; i += (uint64_t)gridDim.x * blockDim.x) dep[i] *= factor;
}

cudaError_t launch_dep_rebase(double *dep, uint64_t cells2, double factor, cudaStream_t st)
{
    int blocks = (int)((cells2 + 255) / 256 < 148 * 8 ? (cells2 + 255) / 256 : 148 * 8);
    dep_rebase_kernel<<<blocks < 1 ? 1 : blocks, 256, 0, st>>>(dep, cells2, factor);
    return cudaGetLastError();
}

// airborne activity in q units: out2[k] += sum of q_k over active slots
__global__ void __launch_bounds__(256) airborne_kernel(const float4 *__restrict__ xyzq, const float *__restrict__ q1, uint64_t n_host,
                                                       const uint64_t *n_dev, int K, double *out2)
{
    __shared__ double s_part[8][2];
    const uint64_t n = n_dev ? *n_dev : n_host;
    double a0 = 0.0, a1 = 0.0;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (uint64_t)gridDim.x * blockDim.x) {
        const float4 p = xyzq[i];
        if (p.z >= 0.0f) {
            a0 += (double)p.w;
            if (K > 1) a1 += (double)q1[i];
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        a0 += __shfl_xor_sync(0xffffffffu, a0, o);
        a1 += __shfl_xor_sync(0xffffffffu, a1, o);
    }
    if ((threadIdx.x & 31) == 0) { s_part[threadIdx.x >> 5][0] = a0; s_part[threadIdx.x >> 5][1] = a1; }
    __syncthreads();
    if (threadIdx.x < 2) {
        double s = 0.0;
        for (int w = 0; w < 8; ++w) s += s_part[w][threadIdx.x];
        if (s != 0.0) atomicAdd(out2 + threadIdx.x, s);
    }
}

cudaError_t launch_airborne(const float4 *xyzq, const float *q1, uint64_t n, const uint64_t *n_dev, int K, double *out2, cudaStream_t st)
{
    airborne_kernel<<<148 * 4, 256, 0, st>>>(xyzq, q1, n, n_dev, K, out2);
    return cudaGetLastError();
}

// export: decode the in-band exit marker (z' = -1 - z) into a status byte
// status 1 = left the domain (ABSORB), 2 = deposited everything it carried (Bernoulli deposition, R11)
__global__ void export_kernel(const float4 *__restrict__ xyzq, const float *__restrict__ q1, uint64_t n_host, const uint64_t *n_dev, float4 *out,
                              uint8_t *status)
{
    const uint64_t n = n_dev ? *n_dev : n_host;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (uint64_t)gridDim.x * blockDim.x) {
        float4 p = xyzq[i];
        uint8_t s = 0;
        if (p.z < 0.0f) { p.z = -1.0f - p.z; s = (p.w == 0.0f && (!q1 || q1[i] == 0.0f)) ? 2 : 1; }
        if (out) out[i] = p;
        if (status) status[i] = s;
    }
}

cudaError_t launch_export(const float4 *xyzq, const float *q1, uint64_t n, const uint64_t *n_dev, float4 *out, uint8_t *status, cudaStream_t st)
{
    export_kernel<<<148 * 4, 256, 0, st>>>(xyzq, q1, n, n_dev, out, status);
    return cudaGetLastError();
}

__global__ void import_kernel(float4 *xyzq, uint64_t n, const uint8_t *status)
{
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (uint64_t)gridDim.x * blockDim.x)
        if (status[i]) xyzq[i].z = -1.0f - xyzq[i].z;
}

cudaError_t launch_import(float4 *xyzq, uint64_t n, const uint8_t *status, cudaStream_t st)
{
    import_kernel<<<148 * 4, 256, 0, st>>>(xyzq, n, status);
    return cudaGetLastError();
}

__global__ void iota_kernel(uint32_t *pid, uint64_t n)
{
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (uint64_t)gridDim.x * blockDim.x)
        pid[i] = (uint32_t)i;
}

cudaError_t launch_iota(uint32_t *pid, uint64_t n, cudaStream_t st)
{
    iota_kernel<<<148 * 4, 256, 0, st>>>(pid, n);
    return cudaGetLastError();
}

// largest stored q per nuclide (lpm_set_particles: bound of the fixed-point deposit scale); q >= 0, so
// the order of the float bit patterns is the order of the values
__global__ void qmax_kernel(const float4 *__restrict__ xyzq, const float *__restrict__ q1, uint64_t n, int K, float *out2)
{
    float m0 = 0.f, m1 = 0.f;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (uint64_t)gridDim.x * blockDim.x) {
        m0 = fmaxf(m0, xyzq[i].w);
        if (K > 1) m1 = fmaxf(m1, q1[i]);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        m0 = fmaxf(m0, __shfl_xor_sync(0xffffffffu, m0, o));
        m1 = fmaxf(m1, __shfl_xor_sync(0xffffffffu, m1, o));
    }
    if ((threadIdx.x & 31) == 0) {
        atomicMax((unsigned int *)out2, __float_as_uint(m0));
        atomicMax((unsigned int *)out2 + 1, __float_as_uint(m1));
    }
}

cudaError_t launch_qmax(const float4 *xyzq, const float *q1, uint64_t n, int K, float *out2, cudaStream_t st)
{
    qmax_kernel<<<148 * 4, 256, 0, st>>>(xyzq, q1, n, K, out2);
    return cudaGetLastError();
}

// ------------------------------------------------------------------ stand-alone parity kernels
__global__ void test_philox_kernel(uint32_t seed_lo, uint32_t seed_hi, uint32_t step, uint32_t stream, uint64_t pid0, uint64_t n, uint32_t *out)
{
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (uint64_t)gridDim.x * blockDim.x) {
        const uint64_t pid = pid0 + i;
        const uint4 r = philox4x32_10(step, stream, (uint32_t)pid, (uint32_t)(pid >> 32), seed_lo, seed_hi);
        out[4 * i] = r.x; out[4 * i + 1] = r.y; out[4 * i + 2] = r.z; out[4 * i + 3] = r.w;
    }
}

cudaError_t launch_test_philox(uint64_t seed, uint64_t step, uint32_t stream, uint64_t pid0, uint64_t n, uint32_t *out, cudaStream_t st)
{
    test_philox_kernel<<<148, 256, 0, st>>>((uint32_t)seed, (uint32_t)(seed >> 32), (uint32_t)step, stream, pid0, n, out);
    return cudaGetLastError();
}

// SURVEY.md 8(c) P1, independent cross-check: NVIDIA's own device Philox4x32-10 (cuRAND, header-only device API)
// with seed -> key, subsequence -> (ctr.z, ctr.w) = particle id, offset / 4 -> (ctr.x, ctr.y) = step.  Test only.
__global__ void test_curand_philox_kernel(uint64_t seed, uint64_t step, uint64_t pid0, uint64_t n, uint32_t *out)
{
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (uint64_t)gridDim.x * blockDim.x) {
        curandStatePhilox4_32_10_t st;
        curand_init((unsigned long long)seed, (unsigned long long)(pid0 + i), (unsigned long long)(4 * step), &st);
        const uint4 r = curand4(&st);
        out[4 * i] = r.x; out[4 * i + 1] = r.y; out[4 * i + 2] = r.z; out[4 * i + 3] = r.w;
    }
}

cudaError_t launch_test_curand_philox(uint64_t seed, uint64_t step, uint64_t pid0, uint64_t n, uint32_t *out, cudaStream_t st)
{
    test_curand_philox_kernel<<<148, 256, 0, st>>>(seed, step, pid0, n, out);
    return cudaGetLastError();
}

__global__ void test_normals_kernel(uint32_t seed_lo, uint32_t seed_hi, uint32_t step, uint64_t pid0, uint64_t n, float *out)
{
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (uint64_t)gridDim.x * blockDim.x) {
        const uint64_t pid = pid0 + i;
        const uint4 r = philox4x32_10(step, 0u, (uint32_t)pid, (uint32_t)(pid >> 32), seed_lo, seed_hi);
        float n0, n1, n2;
        normals3(r, n0, n1, n2);
        out[3 * i] = n0; out[3 * i + 1] = n1; out[3 * i + 2] = n2;
    }
}

cudaError_t launch_test_normals(uint64_t seed, uint64_t step, uint64_t pid0, uint64_t n, float *out, cudaStream_t st)
{
    test_normals_kernel<<<148, 256, 0, st>>>((uint32_t)seed, (uint32_t)(seed >> 32), (uint32_t)step, pid0, n, out);
    return cudaGetLastError();
}

__global__ void test_box_muller_kernel(const uint4 *__restrict__ r, uint64_t n, float *out)
{
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (uint64_t)gridDim.x * blockDim.x) {
        float n0, n1, n2;
        normals3(r[i], n0, n1, n2);
        out[3 * i] = n0; out[3 * i + 1] = n1; out[3 * i + 2] = n2;
    }
}

cudaError_t launch_test_box_muller(const uint32_t *r, uint64_t n, float *out, cudaStream_t st)
{
    test_box_muller_kernel<<<148 * 8, 256, 0, st>>>((const uint4 *)r, n, out);
    return cudaGetLastError();
}

__global__ void test_sample_kernel(const float4 *blend, const __grid_constant__ GridF mg, float kz_min, const float4 *xyz, uint64_t n, float4 *out)
{
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (uint64_t)gridDim.x * blockDim.x) {
        const float4 p = xyz[i];
        const Corner c = mg.nlev ? corner_of<true>(mg, p.x, p.y, p.z) : corner_of<false>(mg, p.x, p.y, p.z);
        float4 m = trilinear(blend, c, mg);   // the step kernel's sampling of a blended buffer
        m.w = fmaxf(m.w, kz_min);
        out[i] = m;
    }
}

cudaError_t launch_test_sample(const float4 *blend, GridF mg, float kz_min, const float4 *xyz, uint64_t n, float4 *out,
                               cudaStream_t st)
{
    test_sample_kernel<<<148, 256, 0, st>>>(blend, mg, kz_min, xyz, n, out);
    return cudaGetLastError();
}

}  // namespace lpm
