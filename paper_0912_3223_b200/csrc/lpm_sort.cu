// lpm_sort.cu — gather-locality pass of the step (pulled into the hot path).
//
// The particle store stays in particle-id order (slot l <-> id, R9), but every 32 to 64 model steps the
// slots are listed in order of the MET CELL their particle sits in (counting sort of 4-byte slot
// indices: histogram -> exclusive scan -> scatter).  The step kernel then walks that list, so the
// 32 lanes of a warp sample the same or neighbouring texels and the texels stay in L1.  What that buys, as
// measured (profiles/r02_c4_step_kernel_ncu.md): a 32-byte gather request of a warp touches about 19 distinct
// sectors in about 5 distinct 128-byte lines and costs about 22 L1 wavefronts - the lanes of a warp are neighbours, not
// twins, so the gathers are NOT down to one or two wavefronts; the gain is the L1 hit rate and the line count.
// Only indices move; the 16-24 B particle records are read and written in place (a scattered 16 B access per
// particle per launch of up to 16 fused steps).  The paper relied on the texture cache for locality (P:L110,
// P:L148); this is its sm_100a counterpart.
#include "lpm_device.cuh"

namespace lpm {

constexpr int kScanItems = 16;                       // items per thread in the scan kernels
constexpr int kScanBlock = 256 * kScanItems;         // items per block

// pass 1: key = offset of the LOWER CORNER texel (i0, j0, k0) of the particle's trilinear stencil in
// the sampled met buffer (the "dual cell"), computed by the same corner_of() the gather uses:
// particles with equal keys read exactly the same eight texels, so a warp of equal keys costs one
// L1 sector per gather instruction instead of one per lane (the L1 data pipe delivers one 32-byte
// sector per cycle; with keys by containing cell a warp still spans the 8 octants = up to 8 lower
// corners).  Exited slots go to the last bucket, n_keys - 1.
__global__ void __launch_bounds__(256) sort_key_kernel(const float4 *__restrict__ xyzq, uint64_t n, const __grid_constant__ GridF g, uint32_t n_keys,
                                                       uint32_t *__restrict__ keys, uint32_t *__restrict__ hist,
                                                       const uint64_t *__restrict__ n_dev = nullptr)
{
    if (n_dev) n = *n_dev;  // (n is a by-value parameter: a local copy)
    // lanes of a warp that share a key count with ONE atomic: next to the source thousands of particles share a
    // cell, and same-address atomics are served at only ~6.5e8/s
    const uint64_t n_round = (n + 31) & ~(uint64_t)31;
    const int lane = threadIdx.x & 31;
    for (uint64_t l = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; l < n_round; l += (uint64_t)gridDim.x * blockDim.x) {
        const bool live = l < n;
        uint32_t key = 0xffffffffu;
        if (live) {
            const float4 p = xyzq[l];
            key = n_keys - 1;
            if (p.z >= 0.0f) key = g.nlev ? corner_of<true>(g, p.x, p.y, p.z).o : corner_of<false>(g, p.x, p.y, p.z).o;
            keys[l] = key;
        }
        const uint32_t peers = __match_any_sync(0xffffffffu, key);
        if (live && lane == __ffs(peers) - 1) atomicAdd(hist + key, (uint32_t)__popc(peers));
    }
}

// pass 2: exclusive scan of hist[0..m) in place: block totals -> scan of the totals -> rescan
__device__ __forceinline__ uint32_t block_exclusive_scan(uint32_t v, uint32_t *s_warp, uint32_t &total)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) s_warp[warp] = inc;
    __syncthreads();
    uint32_t woff = 0, tot = 0;
#pragma unroll
    for (int w = 0; w < 8; ++w) {
        const uint32_t t = s_warp[w];
        woff += w < warp ? t : 0u;
        tot += t;
    }
    __syncthreads();
    total = tot;
    return woff + inc - v;
}

__global__ void __launch_bounds__(256) scan_totals_kernel(const uint32_t *__restrict__ hist, uint32_t m, uint32_t *__restrict__ partial)
{
    __shared__ uint32_t s_warp[8];
    const uint32_t base = blockIdx.x * kScanBlock + threadIdx.x * kScanItems;
    uint32_t s = 0;
#pragma unroll
    for (int i = 0; i < kScanItems; ++i) s += base + i < m ? hist[base + i] : 0u;
    uint32_t total;
    block_exclusive_scan(s, s_warp, total);
    if (threadIdx.x == 0) partial[blockIdx.x] = total;
}

__global__ void __launch_bounds__(256) scan_partials_kernel(uint32_t *partial, uint32_t nb)
{
    __shared__ uint32_t s_warp[8];
    uint32_t carry = 0;
    for (uint32_t b0 = 0; b0 < nb; b0 += 256) {
        const uint32_t i = b0 + threadIdx.x;
        const uint32_t v = i < nb ? partial[i] : 0u;
        uint32_t total;
        const uint32_t ex = block_exclusive_scan(v, s_warp, total);
        if (i < nb) partial[i] = carry + ex;
        carry += total;
    }
}

// live_out (may be null): receives the exclusive offset of the LAST key (the bucket of the exited slots) = the number
// of live particles listed; the scatter pass does not list the exited ones at all
__global__ void __launch_bounds__(256) scan_apply_kernel(uint32_t *__restrict__ hist, uint32_t m, const uint32_t *__restrict__ partial,
                                                         uint64_t *__restrict__ live_out)
{
    __shared__ uint32_t s_warp[8];
    const uint32_t base = blockIdx.x * kScanBlock + threadIdx.x * kScanItems;
    uint32_t v[kScanItems], s = 0;
#pragma unroll
    for (int i = 0; i < kScanItems; ++i) { v[i] = base + i < m ? hist[base + i] : 0u; s += v[i]; }
    uint32_t total;
    uint32_t run = partial[blockIdx.x] + block_exclusive_scan(s, s_warp, total);
#pragma unroll
    for (int i = 0; i < kScanItems; ++i) {
        if (base + i < m) hist[base + i] = run;
        if (live_out && base + i == m - 1) *live_out = run;
        run += v[i];
    }
}

// pass 3: scatter slot indices; lanes of a warp that share a key claim their range with one atomic.
// keys[pos] belongs to the slot list_old[pos] (pos < *live_old, the live length of the previous list: the keys were
// written in the order of that list by the step kernel, so neighbours in `pos` are neighbours in space: the atomics
// aggregate and the writes to the new list fall into a few lines per warp), or to slot pos (pos >= n_old: the
// particles born behind the previous list; no previous list: every pos).  Positions [*live_old, n_old) hold nothing
// (slots that had left the domain before the previous sort are not listed any more).  Slots whose key is the last one
// (exited) are not listed: the new list has hist[n_keys - 1] entries, exported by scan_apply_kernel.
__global__ void __launch_bounds__(256) sort_scatter_kernel(const uint32_t *__restrict__ keys, uint64_t n, uint32_t dead_key, uint32_t *__restrict__ offs,
                                                           const uint32_t *__restrict__ list_old, uint64_t n_old, const uint64_t *__restrict__ live_old,
                                                           uint32_t *__restrict__ perm)
{
    const uint64_t n_round = (n + 31) & ~(uint64_t)31;
    const int lane = threadIdx.x & 31;
    uint64_t n_live_old = n_old;
    if (list_old && live_old) { const uint64_t d = *live_old; n_live_old = d < n_old ? d : n_old; }
    for (uint64_t l = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; l < n_round; l += (uint64_t)gridDim.x * blockDim.x) {
        bool live = l < n && !(list_old && l >= n_live_old && l < n_old);
        uint32_t key = live ? keys[l] : 0xffffffffu;
        if (key == dead_key) { live = false; key = 0xffffffffu; }
        const uint32_t slot = (live && list_old && l < n_old) ? list_old[l] : (uint32_t)l;
        const uint32_t peers = __match_any_sync(0xffffffffu, key);
        const int leader = __ffs(peers) - 1;
        uint32_t base = 0;
        if (live && lane == leader) base = atomicAdd(offs + key, (uint32_t)__popc(peers));
        base = __shfl_sync(0xffffffffu, base, leader);
        if (live) perm[base + __popc(peers & ((1u << lane) - 1u))] = slot;
    }
}

// pass 3, compact mode: move the RECORDS (position, activities, id) instead of listing indices: the
// store itself ends up in dual-cell order (the id travels with the particle there), so the step
// kernel streams it coalesced and consecutive tiles are spatial neighbours.  Order inside a key is
// whatever the atomics give; per-particle results do not depend on storage order (Philox is keyed
// by the id).
__global__ void __launch_bounds__(256) sort_scatter_records_kernel(const uint32_t *__restrict__ keys, const uint64_t *__restrict__ n_dev,
                                                                   uint32_t *__restrict__ offs, const float4 *__restrict__ xyzq,
                                                                   const float *__restrict__ q1, const uint32_t *__restrict__ pid,
                                                                   float4 *__restrict__ xyzq_o, float *__restrict__ q1_o,
                                                                   uint32_t *__restrict__ pid_o)
{
    const uint64_t n = *n_dev;
    const uint64_t n_round = (n + 31) & ~(uint64_t)31;
    const int lane = threadIdx.x & 31;
    for (uint64_t l = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; l < n_round; l += (uint64_t)gridDim.x * blockDim.x) {
        const bool live = l < n;
        const uint32_t key = live ? keys[l] : 0xffffffffu;
        const uint32_t peers = __match_any_sync(0xffffffffu, key);
        const int leader = __ffs(peers) - 1;
        uint32_t base = 0;
        if (live && lane == leader) base = atomicAdd(offs + key, (uint32_t)__popc(peers));
        base = __shfl_sync(0xffffffffu, base, leader);
        if (live) {
            const uint32_t d = base + __popc(peers & ((1u << lane) - 1u));
            xyzq_o[d] = xyzq[l];
            if (q1) q1_o[d] = q1[l];
            pid_o[d] = pid[l];
        }
    }
}

__global__ void __launch_bounds__(256) copy_records_kernel(const uint64_t *__restrict__ n_dev, const float4 *__restrict__ xyzq,
                                                           const float *__restrict__ q1, const uint32_t *__restrict__ pid,
                                                           float4 *__restrict__ xyzq_o, float *__restrict__ q1_o, uint32_t *__restrict__ pid_o)
{
    const uint64_t n = *n_dev;
    for (uint64_t l = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; l < n; l += (uint64_t)gridDim.x * blockDim.x) {
        xyzq_o[l] = xyzq[l];
        if (q1) q1_o[l] = q1[l];
        pid_o[l] = pid[l];
    }
}

// ------------------------------------------------------------------ unordered compaction (B7)
// After a step in hole-list mode: n = ctrl[0] slots, h = ctrl[4] of them listed in holes[] (their particles
// left the domain).  The new count is n - h; every listed hole below it receives a live record from the tail
// [n - h, n) - there are exactly as many of the one as of the other.  Work is proportional to h.
__global__ void __launch_bounds__(256) fill_collect_kernel(const float4 *__restrict__ xyzq, uint64_t *ctrl, const uint32_t *__restrict__ holes,
                                                           uint32_t *__restrict__ src, uint32_t *__restrict__ dst)
{
    const uint64_t n = ctrl[0], h = ctrl[4], new_n = n - h;
    const uint64_t gtid = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x, gstride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t j = gtid; j < h; j += gstride) {
        const uint32_t idx = holes[j];
        if (idx < new_n) dst[atomicAdd((unsigned long long *)(ctrl + 6), 1ull)] = idx;   // a hole that must be filled
        const uint64_t i = new_n + j;                                                     // the j-th slot of the tail
        if (xyzq[i].z >= 0.0f) src[atomicAdd((unsigned long long *)(ctrl + 5), 1ull)] = (uint32_t)i;   // a live record that must move
    }
    if (gtid == 0) ctrl[2] = new_n;
}

__global__ void __launch_bounds__(256) fill_move_kernel(float4 *__restrict__ xyzq, float *__restrict__ q1, uint32_t *__restrict__ pid,
                                                        const uint64_t *__restrict__ ctrl, const uint32_t *__restrict__ src,
                                                        const uint32_t *__restrict__ dst)
{
    const uint64_t cnt = ctrl[5];   // == ctrl[6]
    for (uint64_t j = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; j < cnt; j += (uint64_t)gridDim.x * blockDim.x) {
        const uint32_t s = src[j], d = dst[j];
        xyzq[d] = xyzq[s];
        if (q1) q1[d] = q1[s];
        pid[d] = pid[s];
    }
}

cudaError_t launch_fill_holes(float4 *xyzq, float *q1, uint32_t *pid, uint64_t *ctrl, const uint32_t *holes, uint32_t *src, uint32_t *dst,
                              cudaStream_t st)
{
    fill_collect_kernel<<<sm_count(), 256, 0, st>>>(xyzq, ctrl, holes, src, dst);
    fill_move_kernel<<<sm_count(), 256, 0, st>>>(xyzq, q1, pid, ctrl, src, dst);
    return cudaGetLastError();
}

// compact mode: physical sort of the live records [0, *n_dev) by dual cell, through the alternate
// buffers and back
cudaError_t launch_sort_records(float4 *xyzq, float *q1, uint32_t *pid, const uint64_t *n_dev, uint64_t capacity, GridF g, uint32_t *keys,
                                uint32_t *hist, uint32_t *partial, float4 *xyzq_alt, float *q1_alt, uint32_t *pid_alt, cudaStream_t st)
{
    const uint32_t n_keys = (uint32_t)g.nx * g.ny * g.nz + 1u, m = n_keys;
    cudaError_t e = cudaMemsetAsync(hist, 0, 4ull * n_keys, st);
    if (e != cudaSuccess) return e;
    const uint64_t want = (capacity + 255) / 256, cap = (uint64_t)sm_count() * 8;
    const int blocks = (int)(want < cap ? (want ? want : 1) : cap);
    sort_key_kernel<<<blocks, 256, 0, st>>>(xyzq, 0, g, n_keys, keys, hist, n_dev);
    const uint32_t nb = (m + kScanBlock - 1) / kScanBlock;
    scan_totals_kernel<<<nb, 256, 0, st>>>(hist, m, partial);
    scan_partials_kernel<<<1, 256, 0, st>>>(partial, nb);
    scan_apply_kernel<<<nb, 256, 0, st>>>(hist, m, partial, nullptr);
    sort_scatter_records_kernel<<<blocks, 256, 0, st>>>(keys, n_dev, hist, xyzq, q1, pid, xyzq_alt, q1_alt, pid_alt);
    copy_records_kernel<<<blocks, 256, 0, st>>>(n_dev, xyzq_alt, q1_alt, pid_alt, xyzq, q1, pid);
    return cudaGetLastError();
}

// passes 2 + 3 on keys and a histogram that are already there (written by sort_key_kernel, or by the
// step kernel itself at the end of the launch that precedes a sort)
cudaError_t launch_sort_finish(const uint32_t *keys, uint64_t n, uint32_t n_keys, uint32_t *hist, uint32_t *partial, const uint32_t *list_old,
                               uint64_t n_old, const uint64_t *live_old, uint32_t *perm, uint64_t *live_out, cudaStream_t st)
{
    const uint32_t m = n_keys;
    const uint64_t want = (n + 255) / 256, cap = (uint64_t)sm_count() * 8;
    const int blocks = (int)(want < cap ? (want ? want : 1) : cap);
    const uint32_t nb = (m + kScanBlock - 1) / kScanBlock;
    scan_totals_kernel<<<nb, 256, 0, st>>>(hist, m, partial);
    scan_partials_kernel<<<1, 256, 0, st>>>(partial, nb);
    scan_apply_kernel<<<nb, 256, 0, st>>>(hist, m, partial, live_out);
    sort_scatter_kernel<<<blocks, 256, 0, st>>>(keys, n, n_keys - 1u, hist, list_old, list_old ? n_old : 0, live_old, perm);
    return cudaGetLastError();
}

cudaError_t launch_sort_by_cell(const float4 *xyzq, uint64_t n, GridF g, uint32_t *keys, uint32_t *hist, uint32_t *partial,
                                uint32_t *perm, uint64_t *live_out, cudaStream_t st)
{
    const uint32_t n_keys = (uint32_t)g.nx * g.ny * g.nz + 1u;
    cudaError_t e = cudaMemsetAsync(hist, 0, 4ull * n_keys, st);
    if (e != cudaSuccess) return e;
    const uint64_t want = (n + 255) / 256, cap = (uint64_t)sm_count() * 8;
    const int blocks = (int)(want < cap ? (want ? want : 1) : cap);
    sort_key_kernel<<<blocks, 256, 0, st>>>(xyzq, n, g, n_keys, keys, hist);
    return launch_sort_finish(keys, n, n_keys, hist, partial, nullptr, 0, nullptr, perm, live_out, st);
}

uint64_t sort_partial_entries(uint64_t n_cells) { return (n_cells + 1 + kScanBlock - 1) / kScanBlock + 1; }

}  // namespace lpm
