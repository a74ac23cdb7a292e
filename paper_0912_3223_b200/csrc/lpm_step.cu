// lpm_step.cu — the fused per-particle step kernels for sm_100a.
//
// One thread carries one particle through m >= 1 model steps with its state in registers:
//   a1 Philox4x32-10 + Box-Muller      (R1-R3)
//   a0 the met field of every fused step is blended in time once per launch (blend_kernel below)
//   a2 trilinear gathers of float4 (u,v,w,Kz) from that step's z-fastest buffer (R4)
//   a3 advection + random walk          (R5; Eq.(1)(2))
//   a4 reflection, lateral boundary     (R6, R7)
//   a5 decay / dry / wet deposition     (R8)
//   a6 deposit scatter into the 2-D map (CTA-private fixed-point table in shared memory, then fp64 RED)
//   a7 stable in-place compaction by a single-pass decoupled look-back scan (compact mode)
// The paper's kernel staged particle state in shared memory and sampled hardware textures
// (P:L110-114); neither survives on B200: there is no reuse to stage, and texture filtering's
// fixed-point weights cannot meet the 1e-5 parity bar.
//
// Bounding experiments (profiles/r02_*; NOT part of the product, results are wrong with either):
//   nvcc ... -DLPM_BOUND_NO_DEPOSIT   the step without the deposit scatter a6 (the ledger is still kept)
//   nvcc ... -DLPM_BOUND_NO_GATHER    the step with the eight met texels replaced by values made up in registers (no gathers)
// build a library with one of them next to the product:  nvcc <flags of build.py> -D... -c csrc/lpm_step.cu, link with the other objects.
#include <type_traits>

#include "lpm_device.cuh"

namespace lpm {

template <int K>
struct Acc {  // per-thread ledger partial sums, in activity units before the per-nuclide scale
    float dry[K], wet[K], dec[K];
    float both[K];  // steps where the dry and the decay ledger see the same activity (uniform dry / no sink, no rain)
    float off[K];   // deposit that fell off the map (activity)
};

// a6 deposit scatter, CTA-privatised (S§8(a) a6 "privatised reduce"): the particles of a tile are
// spatial neighbours (gather-locality order), so over the fused steps of a launch their deposits
// fall into a few hundred map cells.  Each CTA sums them in a 1024-slot open-addressing table in
// shared memory keyed by the map cell and sends ONE fp64 RED per touched cell and nuclide to the
// L2-resident map when the tile is done, instead of one per particle-step.
// The sums are FIXED-POINT integers: increment -> rint(inc * S_k), S_k = 2^20 / (largest possible
// increment) rounded down to a power of two, added with the native 32-bit shared atomic (ATOMS.ADD;
// fp32 and 64-bit shared atomics are CAS loops on sm_100).  At most kStepThreads * kMaxFused = 2^12
// increments < 2^20 meet in a slot per tile, so a slot cannot overflow; integer addition is
// associative, so a tile's sums do not depend on the order of the atomics.  Increments in
// [2^17, 2^20) take this path (>= 18 significant bits, round to nearest: relative error <= 1.9e-6
// per increment, unbiased; B4); smaller ones (a particle that carries < 1/8 of the
// largest activity), increments that do not fit and a full table take the direct fp64 RED.
constexpr int kDepSlots = 1024;
static_assert(kStepThreads * kMaxFused <= 4096, "fixed-point deposit sums: 20 bits + 12 bits of count");

// Direct-mapped form of the table: the particles of a tile are spatial neighbours, so their deposits of one launch fall
// into a window of kDepWin x kDepWin map cells around the tile; slot = (cj - wj0) * kDepWin + (ci - wi0), no tags, no
// probing.  The window is centred on the map cell of the tile's first live particle (dep_window, once per tile); a deposit
// outside it (a tile that straddles two rows of the sorted list, an unsorted small ensemble) takes the direct fp64 RED.
constexpr int kDepWin = 32, kDepWinBits = 5, kDepSwz = 5;
static_assert(kDepWin * kDepWin == kDepSlots, "window = table");
template <int K>
struct DepTab {
    int32_t wi0, wj0, ref;
    uint32_t sum[2 * K][kDepSlots];
};

template <int K>
__device__ __forceinline__ void dep_clear(DepTab<K> &T)
{
    for (int i = threadIdx.x; i < kDepSlots; i += kStepThreads) {
#pragma unroll
        for (int k = 0; k < 2 * K; ++k) T.sum[k][i] = 0u;
    }
    if (threadIdx.x == 0) { T.ref = 0x7fffffff; T.wi0 = T.wj0 = 0; }
}

// all threads of the CTA, once per tile before its steps: `live` threads hold a particle at (x, y)
template <int K>
__device__ __forceinline__ void dep_window(const StepArgs &A, DepTab<K> &T, bool live, float x, float y)
{
    if (live) atomicMin(&T.ref, (int32_t)threadIdx.x);
    __syncthreads();
    if ((int32_t)threadIdx.x == T.ref) {
        T.wi0 = __float2int_rd(__fmul_rn(__fsub_rn(x, A.cg.x0), A.cg.inv_dx)) - kDepWin / 2;
        T.wj0 = __float2int_rd(__fmul_rn(__fsub_rn(y, A.cg.y0), A.cg.inv_dy)) - kDepWin / 2;
    }
    __syncthreads();
}

// all threads of the CTA; barriers on both sides belong to the caller
template <int K>
__device__ __forceinline__ void dep_flush(const StepArgs &A, DepTab<K> &T)
{
    const int wi0 = T.wi0, wj0 = T.wj0;
    for (int i = threadIdx.x; i < kDepSlots; i += kStepThreads) {
#pragma unroll
        for (int k = 0; k < K; ++k) {
            const uint32_t vd = T.sum[2 * k][i], vw = T.sum[2 * k + 1][i];
            if (vd | vw) {
                T.sum[2 * k][i] = 0u; T.sum[2 * k + 1][i] = 0u;
                const int dj = i >> kDepWinBits, di = ((i & (kDepWin - 1)) - kDepSwz * dj) & (kDepWin - 1);   // undo the bank swizzle
                const uint32_t cell = (uint32_t)((wj0 + dj) * A.cg.nx + wi0 + di);
                atomicAdd(A.dep + cell + k * A.dep_stride, (double)vd * A.dep_inv_scale[2 * k] + (double)vw * A.dep_inv_scale[2 * k + 1]);
            }
        }
    }
    if (threadIdx.x == 0) T.ref = 0x7fffffff;
}

template <int K>
__device__ __forceinline__ void dep_add(const StepArgs &A, DepTab<K> &T, int slot, uint32_t cell, int k, int w, float v)
{
    const uint32_t iv = __float2uint_rn(v);  // saturating; v >= 0
    if (slot >= 0 && iv - 131072u < 1048576u - 131072u) atomicAdd(&T.sum[w][slot], iv);   // 2^17 <= iv < 2^20: one unsigned compare
    else if (v != 0.0f) atomicAdd(A.dep + cell + k * A.dep_stride, (double)v * A.dep_inv_scale[w]);
}

template <int K, bool WET>
__device__ __forceinline__ void deposit_at(const StepArgs &A, const StepEntry &e, float x, float y, const float (&vd)[K], const float (&vw)[K],
                                           Acc<K> &acc, DepTab<K> &T)
{
    const int ci = cell_of(x, A.cg.x0, A.cg.inv_dx, A.cg.nx);
    const int cj = cell_of(y, A.cg.y0, A.cg.inv_dy, A.cg.ny);
    if ((ci | cj) < 0) {  // off the map: ledger only
#pragma unroll
        for (int k = 0; k < K; ++k) {
            acc.off[k] += vd[k] * e.Oid[k];
            if (WET) acc.off[k] += vw[k] * e.Oiw[k];
        }
        return;
    }
    const uint32_t cell = (uint32_t)(cj * A.cg.nx + ci);
    const uint32_t di = (uint32_t)(ci - T.wi0), dj = (uint32_t)(cj - T.wj0);
    // slot = row dj, column (di + kDepSwz dj) mod 32: the shared-memory bank of a slot is its column, and the particles of
    // a warp cover a block of a few x few map cells - unswizzled, the cells of one map column would share a bank and
    // their atomics be served one after the other (ncu r02a: 8.8 wavefronts per ATOMS, 16 % of the L1 data pipe)
    const int slot = (di | dj) < (uint32_t)kDepWin ? (int)((dj << kDepWinBits) | ((di + kDepSwz * dj) & (kDepWin - 1))) : -1;
#pragma unroll
    for (int k = 0; k < K; ++k) {
        dep_add<K>(A, T, slot, cell, k, 2 * k, vd[k]);
        if (WET) dep_add<K>(A, T, slot, cell, k, 2 * k + 1, vw[k]);
    }
}

// One model step of one particle.  Returns false when the particle left the domain (ABSORB).
// Source order = intended issue order: the eight gathers go out first and the ~150 instructions of
// Philox + Box-Muller run while they are in flight.
template <int K, int DRY, bool BERN, bool EQ3, bool ZLEV, bool ZP = false>
__device__ __forceinline__ bool step_once(const StepArgs &A, const StepEntry &e, uint32_t step_lo,
                                          uint32_t pid_lo, float &x, float &y, float &z,
                                          float (&q)[K], Acc<K> &acc, DepTab<K> &dep)
{
    // a0 + a2: weather at X_old, t_n
    Corner c = corner_of<ZLEV>(A.mg, x, y, z);
    float dkz = 0.0f;  // drift-corrected walk (labelled departure): dKz/dz of the sampled field
    const uint32_t o_cell = c.o;
    c.o += e.buf * (uint32_t)A.snap_cells;   // texel index inside the whole set of blended buffers (< 2^32: lpm_create)
    const float4 m = trilinear<ZP>(A.blend, c, A.mg, ZLEV && A.drift != 0, &dkz);
    c.o = o_cell;
    // Kz: the interpolated gridded field (R4), or Eq.(3) per particle from the 2-D fields of this step (R12)
    const float kz = fmaxf(EQ3 ? kz_eq3(A.surf + (uint64_t)e.buf * (uint32_t)(A.mg.nx * A.mg.ny), c, A.mg, z) : m.w, A.kz_min);

    // a1: three N(0,1) from Philox stream 0
    const uint4 r = philox4x32_10_rk<0u>(step_lo, pid_lo, A.rk);
    float n0, n1, n2;
    normals3(r, n0, n1, n2);

    // a3: Eq.(1) + Eq.(2)
    x = fmaf(A.sigma_h, n0, fmaf(m.x, A.dt, x));
    y = fmaf(A.sigma_h, n1, fmaf(m.y, A.dt, y));
    z = fmaf(sqrt_nr(2.0f * A.dt * kz), n2, fmaf(m.z, A.dt, z));
    if (ZLEV && A.drift && !(m.w < A.kz_min)) z = fmaf(dkz, A.dt, z);  // (a floored Kz is constant in z)

    // a4: reflection (R6), lateral boundary (R7)
    z = fabsf(z);
    if (z > A.H) z = 2.0f * A.H - z;
    z = fmaxf(z, 0.0f);
    if (A.absorb) {
        const bool inside = (x >= A.bx0) & (x < A.bx1) & (y >= A.by0) & (y < A.by1);
        if (!inside) {
#pragma unroll
            for (int k = 0; k < K; ++k) atomicAdd(A.ledger + k * 8 + 5, (double)q[k] * e.G[k]);
            return false;
        }
    }

    // a5: deposition then decay at the new position (R8).  Activity = q * G_k(t_n); decay and
    // uniform dry loss live in G, so q only changes for position-dependent sinks.  DRY is a
    // template parameter and the rain flag is the same for every thread, so the common cases are
    // straight-line code: no sink at all (2 FMA), uniform dry deposition without rain (4 FMA + the
    // scatter).
    const bool raining = (e.snap >> 16) & 1;
    if constexpr (BERN) {
        // R11, the paper's own form: one Bernoulli trial per nuclide and sink per step from
        // Philox stream 1; u = (word >> 8) 2^-24 < p decides (exact on both sides); an event deposits the
        // nuclide's whole activity at the new (x, y) - a rare event, so straight to the map with an fp64 RED;
        // a particle that carries nothing any more becomes inactive.
        const bool dry_here = DRY == kDryUniform || (DRY == kDryLayer && z < A.h_dep);
        const bool wet_here = raining & (x >= A.rx0) & (x < A.rx1) & (y >= A.ry0) & (y < A.ry1);
        if (dry_here | wet_here) {
            const uint4 r1 = philox4x32_10_rk<1u>(step_lo, pid_lo, A.rk);
            const uint32_t wd[2] = {r1.x, r1.y}, ww[2] = {r1.z, r1.w};
            constexpr float s24 = 5.9604644775390625e-08f;
#pragma unroll
            for (int k = 0; k < K; ++k) {
                if (q[k] > 0.0f) {
                    const bool d = dry_here && __uint2float_rn(wd[k] >> 8) * s24 < A.p_dry[k];
                    const bool w = !d && wet_here && __uint2float_rn(ww[k] >> 8) * s24 < A.p_wet[k];
                    if (d | w) {
                        const double act = (double)q[k] * e.G[k];
                        const int ci = cell_of(x, A.cg.x0, A.cg.inv_dx, A.cg.nx);
                        const int cj = cell_of(y, A.cg.y0, A.cg.inv_dy, A.cg.ny);
                        if ((ci | cj) >= 0) atomicAdd(A.dep + (uint32_t)(cj * A.cg.nx + ci) + k * A.dep_stride, act * e.Eg[k]);
                        else atomicAdd(A.ledger + k * 8 + 6, act);
                        atomicAdd(A.ledger + k * 8 + (d ? 2 : 3), act);
                        q[k] = 0.0f;
                    }
                }
            }
        }
        bool empty = true;
#pragma unroll
        for (int k = 0; k < K; ++k) {
            acc.both[k] = fmaf(q[k], e.Gf[k], acc.both[k]);
            empty &= !(q[k] > 0.0f);
        }
        return !empty;
    }
    if (DRY != kDryLayer && !raining) {
#pragma unroll
        for (int k = 0; k < K; ++k) acc.both[k] = fmaf(q[k], e.Gf[k], acc.both[k]);
        if constexpr (DRY != kDryNone) {
            float vd[K];
#pragma unroll
            for (int k = 0; k < K; ++k) vd[k] = q[k] * e.Gps[k];
#ifndef LPM_BOUND_NO_DEPOSIT
            deposit_at<K, false>(A, e, x, y, vd, vd, acc, dep);
#endif
        }
        return true;
    }
    const bool dry_here = DRY == kDryUniform || (DRY == kDryLayer && z < A.h_dep);
    const bool wet_here = raining & (x >= A.rx0) & (x < A.rx1) & (y >= A.ry0) & (y < A.ry1);
    float vd[K], vw[K];
#pragma unroll
    for (int k = 0; k < K; ++k) {
        const float G = e.Gf[k];
        float act = q[k] * G;
        vd[k] = 0.0f;
        vw[k] = 0.0f;
        if (dry_here) {
            acc.dry[k] += act;
            if (DRY == kDryLayer) {
                vd[k] = act * e.Pd[k];
                q[k] = fmaf(-q[k], A.p_dry[k], q[k]);
                act = q[k] * G;
            } else {
                vd[k] = q[k] * e.Gps[k];
            }
        }
        if (wet_here) {
            vw[k] = act * e.Pw[k];
            acc.wet[k] += act;
            q[k] = fmaf(-q[k], A.p_wet[k], q[k]);
            act = q[k] * G;
        }
        acc.dec[k] += act;
    }

    // a6: deposit at the cell of the NEW (x, y)
#ifndef LPM_BOUND_NO_DEPOSIT
    if (dry_here | wet_here) deposit_at<K, true>(A, e, x, y, vd, vw, acc, dep);
#endif
    return true;
}

// block-reduce the per-thread ledger partials and add them to the device ledger (one fp64 RED per
// quantity per CTA)
template <int K>
__device__ __forceinline__ void flush_ledger(const StepArgs &A, const Acc<K> &acc)
{
    __shared__ float s_part[kStepThreads / 32][4 * K];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < K; ++k) {
        const float b = warp_sum(acc.both[k]);
        const float d = (A.dry_mode == kDryUniform && !A.bern ? b : 0.0f) + warp_sum(acc.dry[k]), w = warp_sum(acc.wet[k]), c = b + warp_sum(acc.dec[k]), o = warp_sum(acc.off[k]);
        if (lane == 0) { s_part[warp][4 * k] = d; s_part[warp][4 * k + 1] = w; s_part[warp][4 * k + 2] = c; s_part[warp][4 * k + 3] = o; }
    }
    __syncthreads();
    if (threadIdx.x < 4 * K) {
        double s = 0.0;
#pragma unroll
        for (int w = 0; w < kStepThreads / 32; ++w) s += (double)s_part[w][threadIdx.x];
        const int k = threadIdx.x / 4, f = threadIdx.x % 4;
        const double scale = f == 0 ? (double)A.p_dry[k] : (f == 1 ? A.wet_scale[k] : (f == 2 ? A.dec_scale[k] : 1.0));
        if (s != 0.0) atomicAdd(A.ledger + k * 8 + (f == 3 ? 6 : 2 + f), s * scale);
    }
}

// a8 fused into the step (round 2): the launch that ends on a binning step bins its particles while they are still in
// registers - no second pass over the particle store (the stand-alone bin_tile_kernel of lpm_bin.cu reads 12 + 4 K bytes per
// particle again and, walking the store in slot order, finds few particles of a tile in the same cell).  Here the 256
// particles of a tile are spatial neighbours (gather-locality order), so their counts and fixed-point sums meet in a
// CTA-private open-addressing table keyed by the concentration cell - the same table, and the same shared memory, as the
// deposit table, which is idle once the tile's steps are done - and every touched cell receives one RED per field.
constexpr int kBinTabSlots = 1024, kBinTabBits = 10, kBinTabProbes = 8;
template <int K>
struct BinTabS {
    uint32_t tag[kBinTabSlots];      // cell + 1, 0 = empty
    uint32_t cnt[kBinTabSlots];
    uint32_t sum[K][kBinTabSlots];   // rint(q * S_k), S_k = StepArgs::bin_scale
};
template <int K>
union TileTab {
    DepTab<K> dep;
    BinTabS<K> bin;
};

// all threads of the CTA, after the tile's steps and the flush of its deposit table; `live`: this thread holds an active
// particle at (x, y, z) carrying q.  Leaves the shared memory zeroed (= an empty deposit table).
template <int K>
__device__ __forceinline__ uint32_t bin_tile(const StepArgs &A, BinTabS<K> &B, bool live, float x, float y, float z, const float (&q)[K])
{
    __syncthreads();                                   // the deposit table has been flushed: all words are zero ...
    if (threadIdx.x < 4) B.tag[threadIdx.x] = 0u;      // ... except the window header that overlays the first tags
    __syncthreads();
    uint32_t binned = 0;
    if (live) {
        const int ci = cell_of(x, A.cg.x0, A.cg.inv_dx, A.cg.nx);
        const int cj = cell_of(y, A.cg.y0, A.cg.inv_dy, A.cg.ny);
        const int ck = cell_of(z, A.cg.z0, A.cg.inv_dz, A.cg.nz);
        if ((ci | cj | ck) >= 0) {
            binned = 1;
            const uint32_t cell = (uint32_t)((ck * A.cg.ny + cj) * A.cg.nx + ci), key = cell + 1u;
            uint32_t h = (key * 0x9E3779B1u) >> (32 - kBinTabBits);
            int s = -1;
#pragma unroll 1
            for (int pr = 0; pr < kBinTabProbes; ++pr) {
                const uint32_t t = *(volatile uint32_t *)&B.tag[h];
                if (t == key) { s = (int)h; break; }
                if (t == 0u) {
                    const uint32_t old = atomicCAS(&B.tag[h], 0u, key);
                    if (old == 0u || old == key) { s = (int)h; break; }
                }
                h = (h + 1u) & (kBinTabSlots - 1);
            }
            if (s >= 0) atomicAdd(&B.cnt[s], 1u);
            else atomicAdd(A.bin_cnt + cell, 1u);
#pragma unroll
            for (int k = 0; k < K; ++k) {
                const uint32_t iv = __float2uint_rn(q[k] * A.bin_scale[k]);   // saturating; q >= 0
                if (s >= 0 && iv - 131072u < 1048576u - 131072u) atomicAdd(&B.sum[k][s], iv);
                else if (q[k] != 0.0f) atomicAdd(A.bin_conc + (uint64_t)k * A.bin_cells3 + cell, (double)q[k]);
            }
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < kBinTabSlots; i += kStepThreads) {
        const uint32_t key = B.tag[i];
        if (key == 0u) continue;
        B.tag[i] = 0u;
        const uint32_t c = B.cnt[i];
        B.cnt[i] = 0u;
        atomicAdd(A.bin_cnt + (key - 1u), c);
#pragma unroll
        for (int k = 0; k < K; ++k) {
            const uint32_t v = B.sum[k][i];
            B.sum[k][i] = 0u;
            if (v) atomicAdd(A.bin_conc + (uint64_t)k * A.bin_cells3 + (key - 1u), (double)v * A.bin_inv_scale[k]);
        }
    }
    __syncthreads();
    return binned;
}

// ------------------------------------------------------------------ slot-addressed kernel
// Particles of one release occupy the slots base + [0, n); slot l carries global particle id
// pid_offset + l * pid_stride, so ids (and birth steps, R9) are implied by the slot.  Persistent
// grid-stride loop; up to kMaxFused model steps per launch.
#ifndef LPM_STEP_MINB
#define LPM_STEP_MINB 4
#endif
static_assert(sizeof(StepArgs) <= 32764, "StepArgs must fit the kernel-parameter space (32764 B since CUDA 12.1 on sm_70+)");

// BIN: the instantiation for the launch that ends on a binning step (a8 fused; default physics only).  A separate
// instantiation because the epilogue's registers and shared-memory union cost the step loop 5 % when compiled in
// (measured: 7.32e10 -> 6.98e10 particle-steps/s on c4), and 44 of 45 launches do not bin.
template <int K, int DRY, bool BERN, bool EQ3, bool ZLEV, bool ZP = false, bool BIN = false>
__global__ void __launch_bounds__(kStepThreads, LPM_STEP_MINB) step_slots_kernel(const __grid_constant__ StepArgs A)
{
    __shared__ uint32_t s_ticket;
    Acc<K> acc;
#pragma unroll
    for (int k = 0; k < K; ++k) acc.dry[k] = acc.wet[k] = acc.dec[k] = acc.both[k] = acc.off[k] = 0.0f;

    // Dynamic tile schedule in list order: tiles [0, t_old) walk the sorted slot list (particles that
    // existed at the last gather-locality sort, in dual-cell order), tiles [t_old, n_tiles) the
    // younger slots in id order (still close to the source).  The CTAs resident together therefore
    // work on one small region of the plume: their met gathers hit L1/L2, and their deposits meet
    // in the CTA-private tables below instead of in the global map.
    __shared__ typename std::conditional<BIN, TileTab<K>, DepTab<K>>::type U;
    DepTab<K> &T = *reinterpret_cast<DepTab<K> *>(&U);
    if constexpr (BIN) {
        for (int i = threadIdx.x; i < (int)(sizeof(U) / 4); i += kStepThreads) ((uint32_t *)&U)[i] = 0u;
        __syncthreads();
    }
    dep_clear<K>(T);
    __shared__ uint32_t s_binned;   // BIN: particles binned by this CTA (kept in shared memory: no register lives across the step loop)
    if (BIN && threadIdx.x == 0) s_binned = 0u;
    // (slots that had left the domain when the list was built are not on it: its live length is a device scalar)
    uint64_t n_list = A.perm ? A.n_perm : 0ull;
    if (A.perm && A.n_live) { const uint64_t d = *A.n_live; n_list = d < n_list ? d : n_list; }
    const uint32_t t_old = (uint32_t)((n_list + kStepThreads - 1) / kStepThreads);
    const uint64_t first_new = A.perm ? A.n_perm : 0ull;
    const uint32_t n_tiles = t_old + (uint32_t)((A.n - first_new + kStepThreads - 1) / kStepThreads);
    uint32_t n_done = 0;   // particle-steps this thread executed (bench.py's unit: born AND active particles x steps)
    for (;;) {
        __syncthreads();
        if (threadIdx.x == 0) s_ticket = (uint32_t)atomicAdd((unsigned long long *)(A.ctrl + 16), 1ull);
        __syncthreads();
        const uint32_t tile = s_ticket;
        if (tile >= n_tiles) break;
        uint64_t l, pos;   // slot (relative to the release block) and its position in the list
        bool valid;
        if (tile < t_old) {
            pos = (uint64_t)tile * kStepThreads + threadIdx.x;
            valid = pos < n_list;
            l = valid ? A.perm[pos] : 0ull;
        } else {
            l = pos = first_new + (uint64_t)(tile - t_old) * kStepThreads + threadIdx.x;
            valid = l < A.n;
        }
        const bool in_range = valid;
        const uint64_t slot = A.base + l;
        const uint32_t pid = (uint32_t)(A.pid_offset + l * A.pid_stride);
        float x = 0.f, y = 0.f, z = 0.f, q[K];
#pragma unroll
        for (int k = 0; k < K; ++k) q[k] = 0.f;
        int s_begin = 0;
        if (valid) {
            if (l >= A.n_prev) {
                // born inside this launch (R9): count mode b = s_start + floor(j*S/N), rate mode
                // b = s_start + l / c
                const int64_t b = A.rel_N ? A.rel_s_start + (int64_t)(((uint64_t)pid * (uint64_t)A.rel_S) / A.rel_N)
                                          : A.rel_s_start + (int64_t)(l / A.rel_c);
                s_begin = (int)(b - (int64_t)A.step0);
                x = A.sx; y = A.sy; z = A.sz;
#pragma unroll
                for (int k = 0; k < K; ++k) q[k] = (float)(A.emit[k] / A.tab[s_begin].G[k]);
            } else {
                const float4 p = A.xyzq[slot];
                x = p.x; y = p.y; z = p.z; q[0] = p.w;
                if (K > 1) q[1] = A.q1[slot];
                valid = z >= 0.0f;  // z < 0: exited earlier (ABSORB without compaction)
            }
        }
        if (A.any_dep) dep_window<K>(A, T, valid, x, y);
        if (valid) {
            // the trip count is the same for every thread (uniform table index, uniform branches inside
            // the step); a particle born inside this launch or absorbed at the boundary skips steps
            bool alive = true;
            const uint32_t step0 = (uint32_t)A.step0;
            for (int s = 0; s < A.m_steps; ++s)
                if (alive & (s >= s_begin)) {
                    alive = step_once<K, DRY, BERN, EQ3, ZLEV, ZP>(A, A.tab[s], step0 + (uint32_t)s, pid, x, y, z, q, acc, T);
                    ++n_done;
                }
            if (!alive) z = -1.0f - z;  // exit position kept, slot marked inactive
            A.xyzq[slot] = make_float4(x, y, z, q[0]);
            if (K > 1) A.q1[slot] = q[1];
        }
        if (A.mask && valid && z >= 0.0f) {
            // tile of the particle's met column at the end of the launch -> plume mask of the next blend
            const int ci = min(max(__float2int_rd((x - A.mg.x0) * A.mg.inv_dx), 0), A.mg.nx - 1);
            const int cj = min(max(__float2int_rd((y - A.mg.y0) * A.mg.inv_dy), 0), A.mg.ny - 1);
            A.mask[(cj / kMaskTile) * A.mask_ntx + ci / kMaskTile] = 1;
        }
        if (A.keys_out) {
            // pass 1 of the coming gather-locality sort, for free: the new position is in registers; the lanes of
            // a warp that share a key (most of them, in a sorted warp) count with one atomic.  The keys are stored in
            // LIST order (coalesced here, and the scatter pass then walks spatial neighbours: lpm_sort.cu), or by slot
            // for large ensembles (sort row: the slot-order scatter leaves each cell's slots ascending)
            uint32_t key = 0xffffffffu;
            if (in_range) {
                key = (valid && z >= 0.0f) ? corner_of<ZLEV>(A.mg, x, y, z).o : A.n_keys - 1u;
                A.keys_out[A.keys_by_slot ? l : pos] = key;
            }
            const uint32_t peers = __match_any_sync(0xffffffffu, key);
            if (in_range && (threadIdx.x & 31) == __ffs(peers) - 1) atomicAdd(A.hist_out + key, (uint32_t)__popc(peers));
        }
        if (A.any_dep) {
            __syncthreads();
            dep_flush<K>(A, T);
        }
        if constexpr (BIN) {   // this launch ends on a binning step (a8 fused)
            const uint32_t b = bin_tile<K>(A, *reinterpret_cast<BinTabS<K> *>(&U), valid && z >= 0.0f, x, y, z, q);
            const uint32_t bw = __reduce_add_sync(0xffffffffu, b);
            if ((threadIdx.x & 31) == 0 && bw) atomicAdd(&s_binned, bw);
            dep_clear<K>(T);                           // window header of the deposit table (the sums are zero again)
        }
    }
    flush_ledger<K>(A, acc);
    if constexpr (BIN) {
        __syncthreads();
        if (threadIdx.x == 0 && s_binned) atomicAdd((unsigned long long *)(A.ctrl + 19), (unsigned long long)s_binned);
    }
    n_done = __reduce_add_sync(0xffffffffu, n_done);
    if ((threadIdx.x & 31) == 0 && n_done) atomicAdd((unsigned long long *)(A.ctrl + 3), (unsigned long long)n_done);
}

// ------------------------------------------------------------------ compacting kernel (a7)
// One model step with stable in-place stream compaction of the particles that left the domain,
// fused into the store: each 1024-particle tile (4 per thread) steps its particles, counts survivors, obtains its
// exclusive output offset from a single-pass decoupled look-back over the tile states, and
// writes its survivors at [offset, offset + count).  In place is safe: a tile publishes only
// after it has loaded its inputs, and the destination range of tile t lies inside the source
// ranges of tiles <= t, all of which have published (hence loaded) before t learns its offset.
__device__ __forceinline__ uint64_t ld_state(const uint64_t *p)
{
    uint64_t v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_state(uint64_t *p, uint64_t v)
{
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

template <int K, int DRY, bool BERN, bool EQ3, bool ZLEV>
__global__ void __launch_bounds__(kStepThreads) step_compact_kernel(const __grid_constant__ StepArgs A)
{
    constexpr int kItems = kScanTile / kStepThreads;  // particles per thread and tile: amortises the tile's barriers and look-back
    constexpr int kParts = kItems * (kStepThreads / 32);
    __shared__ uint32_t s_tile;
    __shared__ uint32_t s_woff[kParts];  // survivors per (item, warp), then their exclusive offsets in index order
    __shared__ uint32_t s_excl;
    Acc<K> acc;
#pragma unroll
    for (int k = 0; k < K; ++k) acc.dry[k] = acc.wet[k] = acc.dec[k] = acc.both[k] = acc.off[k] = 0.0f;

    const uint64_t n = A.ctrl[0];
    const uint32_t n_tiles = (uint32_t)((n + kScanTile - 1) / kScanTile);
    const uint32_t epoch = ((uint32_t)(A.step0 + 1) & 0x3fffffffu) << 2;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    constexpr uint32_t FLAG_A = 1u, FLAG_P = 2u;
    static_assert(kParts == 32, "the per-tile offsets are scanned by one warp");
    __shared__ DepTab<K> T;
    dep_clear<K>(T);
    __syncthreads();

    for (;;) {
        if (threadIdx.x == 0) s_tile = (uint32_t)atomicAdd((unsigned long long *)(A.ctrl + 1), 1ull);
        __syncthreads();
        const uint32_t tile = s_tile;
        if (tile >= n_tiles) break;

        float x[kItems], y[kItems], z[kItems], q[kItems][K];
        uint32_t pid[kItems], rank[kItems];
        bool alive[kItems];
#pragma unroll
        for (int j = 0; j < kItems; ++j) {
            const uint64_t i = (uint64_t)tile * kScanTile + (uint32_t)j * kStepThreads + threadIdx.x;
            alive[j] = false;
            x[j] = y[j] = z[j] = 0.f;
            pid[j] = 0;
#pragma unroll
            for (int k = 0; k < K; ++k) q[j][k] = 0.f;
            if (i < n) {
                const float4 p = A.xyzq[i];
                x[j] = p.x; y[j] = p.y; z[j] = p.z; q[j][0] = p.w;
                if (K > 1) q[j][1] = A.q1[i];
                pid[j] = A.pid[i];
            }
        }
        if (A.any_dep) dep_window<K>(A, T, (uint64_t)tile * kScanTile + threadIdx.x < n, x[0], y[0]);
#pragma unroll
        for (int j = 0; j < kItems; ++j) {
            const uint64_t i = (uint64_t)tile * kScanTile + (uint32_t)j * kStepThreads + threadIdx.x;
            if (i < n) alive[j] = step_once<K, DRY, BERN, EQ3, ZLEV>(A, A.tab[0], (uint32_t)A.step0, pid[j], x[j], y[j], z[j], q[j], acc, T);
            // survivors: rank inside the (item, warp) part
            const uint32_t ball = __ballot_sync(0xffffffffu, alive[j]);
            rank[j] = __popc(ball & ((1u << lane) - 1u));
            if (lane == 0) s_woff[j * (kStepThreads / 32) + warp] = __popc(ball);
        }
        if (A.holes) {
            // Unordered store (gather_sort on, B7): no scan at all.  Survivors are written back where they
            // are; the slots of the particles that left are listed, and fill_holes_* moves the live records of the
            // tail into the listed holes below the new count (work proportional to the number of exits).
#pragma unroll
            for (int j = 0; j < kItems; ++j) {
                const uint64_t i = (uint64_t)tile * kScanTile + (uint32_t)j * kStepThreads + threadIdx.x;
                const bool dead = i < n && !alive[j];
                if (i < n) {
                    A.xyzq[i] = make_float4(x[j], y[j], alive[j] ? z[j] : -1.0f - z[j], q[j][0]);
                    if (K > 1) A.q1[i] = q[j][1];
                }
                const uint32_t ball = __ballot_sync(0xffffffffu, dead);
                if (ball) {
                    uint32_t base = 0;
                    if (lane == 0) base = (uint32_t)atomicAdd((unsigned long long *)(A.ctrl + 4), (unsigned long long)__popc(ball));
                    base = __shfl_sync(0xffffffffu, base, 0);
                    if (dead) A.holes[base + __popc(ball & ((1u << lane) - 1u))] = (uint32_t)i;
                }
            }
        } else {
            __syncthreads();  // also orders every thread's input loads before the publication below
            if (warp == 0) {
                // exclusive scan of the 32 part counts (index order = item-major), tile total
                const uint32_t cnt = s_woff[lane];
                uint32_t inc = cnt;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
                    if (lane >= o) inc += t;
                }
                s_woff[lane] = inc - cnt;
                const uint32_t total = __shfl_sync(0xffffffffu, inc, 31);
                uint32_t excl = 0;
                if (lane == 0) {
                    __threadfence();
                    st_state(A.tile_state + tile, ((uint64_t)(epoch | (tile == 0 ? FLAG_P : FLAG_A)) << 32) | total);
                }
                if (tile > 0) {
                    // warp-wide look-back: lane l inspects tile (look - l)
                    int look = (int)tile - 1;
                    for (;;) {
                        const int t = look - lane;
                        uint64_t st = 0;
                        uint32_t flag = FLAG_P, val = 0;
                        if (t >= 0) {
                            do { st = ld_state(A.tile_state + t); } while (((uint32_t)(st >> 32) & ~3u) != epoch);
                            flag = (uint32_t)(st >> 32) & 3u;
                            val = (uint32_t)st;
                        }
                        const uint32_t pmask = __ballot_sync(0xffffffffu, flag == FLAG_P);
                        const int first_p = pmask ? __ffs(pmask) - 1 : 31;  // t < 0 lanes count as P with value 0; no P: all 32 aggregates count
                        uint32_t contrib = (lane <= first_p) ? val : 0u;
#pragma unroll
                        for (int o = 16; o > 0; o >>= 1) contrib += __shfl_xor_sync(0xffffffffu, contrib, o);
                        excl += contrib;
                        if (pmask) break;
                        look -= 32;
                    }
                    if (lane == 0) st_state(A.tile_state + tile, ((uint64_t)(epoch | FLAG_P) << 32) | (excl + total));
                }
                if (lane == 0) {
                    s_excl = excl;
                    if (tile == n_tiles - 1) A.ctrl[2] = (uint64_t)excl + total;
                    __threadfence();
                }
            }
            __syncthreads();
#pragma unroll
            for (int j = 0; j < kItems; ++j) {
                if (alive[j]) {
                    const uint64_t dst = (uint64_t)s_excl + s_woff[j * (kStepThreads / 32) + warp] + rank[j];
                    A.xyzq[dst] = make_float4(x[j], y[j], z[j], q[j][0]);
                    if (K > 1) A.q1[dst] = q[j][1];
                    A.pid[dst] = pid[j];
                }
            }
        }
        if (A.mask) {
            // tiles of the survivors' met columns -> plume mask of the next blend
#pragma unroll
            for (int j = 0; j < kItems; ++j) {
                if (alive[j]) {
                    const int ci = min(max(__float2int_rd((x[j] - A.mg.x0) * A.mg.inv_dx), 0), A.mg.nx - 1);
                    const int cj = min(max(__float2int_rd((y[j] - A.mg.y0) * A.mg.inv_dy), 0), A.mg.ny - 1);
                    A.mask[(cj / kMaskTile) * A.mask_ntx + ci / kMaskTile] = 1;
                }
            }
        }
        if (A.any_dep) {
            if (A.holes) __syncthreads();   // the hole-list branch has no barrier of its own: every thread's deposits first
            dep_flush<K>(A, T);             // (scan branch: every thread's step is behind the barriers above)
        }
        __syncthreads();  // s_tile / s_woff / s_excl and the deposit table are reused by the next tile
    }
    flush_ledger<K>(A, acc);
}

// newborn particles of one step, appended behind the live ones (compact mode, R9)
__global__ void __launch_bounds__(256) inject_kernel(const __grid_constant__ InjectArgs A)
{
    const uint64_t n_prev = A.ctrl[2];
    uint64_t running = n_prev;
    const uint64_t gtid = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const uint64_t gstride = (uint64_t)gridDim.x * blockDim.x;
    for (int r = 0; r < A.n_spec; ++r) {
        const InjectSpec &sp = A.spec[r];
        const uint64_t room = A.capacity > running ? A.capacity - running : 0;
        const uint64_t take = sp.count < room ? sp.count : room;  // highest j skipped (R9)
        for (uint64_t j = gtid; j < take; j += gstride) {
            const uint64_t slot = running + j;
            A.xyzq[slot] = make_float4(sp.sx, sp.sy, sp.sz, sp.q[0]);
            if (A.K > 1) A.q1[slot] = sp.q[1];
            A.pid[slot] = (uint32_t)(sp.first_pid + j * sp.pid_stride);
        }
        if (gtid == 0) A.ctrl[8 + sp.rel_index] += take;  // per-release emitted count (ledger)
        running += take;
    }
    if (gtid == 0) {
        A.ctrl[0] = running;
        A.ctrl[1] = 0;
        A.ctrl[4] = 0; A.ctrl[5] = 0; A.ctrl[6] = 0;  // hole list and fill counters of the coming step
        A.ctrl[3] += running;  // cumulative particle-steps (timing hooks)
        if (A.log_slot) *A.log_slot = running - n_prev;
    }
}

// ------------------------------------------------------------------ launchers
typedef void (*StepKernel)(const StepArgs);

// One instantiation per (nuclide count, dry-deposition mode, expected-mass / Bernoulli deposition, gridded / Eq.(3) Kz, uniform / non-uniform levels).
template <int K, bool BERN, bool EQ3, bool ZLEV>
static StepKernel pick_dry(bool compact, int dry)
{
    if (compact) {
        if (dry == kDryNone) return step_compact_kernel<K, kDryNone, BERN, EQ3, ZLEV>;
        return dry == kDryUniform ? step_compact_kernel<K, kDryUniform, BERN, EQ3, ZLEV> : step_compact_kernel<K, kDryLayer, BERN, EQ3, ZLEV>;
    }
    if (dry == kDryNone) return step_slots_kernel<K, kDryNone, BERN, EQ3, ZLEV>;
    return dry == kDryUniform ? step_slots_kernel<K, kDryUniform, BERN, EQ3, ZLEV> : step_slots_kernel<K, kDryLayer, BERN, EQ3, ZLEV>;
}

template <int K, bool BERN>
static StepKernel pick_kb(bool compact, int dry, bool eq3, bool zlev)
{
    if (eq3) return zlev ? pick_dry<K, BERN, true, true>(compact, dry) : pick_dry<K, BERN, true, false>(compact, dry);
    return zlev ? pick_dry<K, BERN, false, true>(compact, dry) : pick_dry<K, BERN, false, false>(compact, dry);
}

// z-pair texels and / or the fused binning epilogue: default physics, slot-addressed store only (18 more instantiations, not 96 x 4)
template <int K, bool ZP, bool BIN>
static StepKernel pick_zp(int dry)
{
    if (dry == kDryNone) return step_slots_kernel<K, kDryNone, false, false, false, ZP, BIN>;
    return dry == kDryUniform ? step_slots_kernel<K, kDryUniform, false, false, false, ZP, BIN> : step_slots_kernel<K, kDryLayer, false, false, false, ZP, BIN>;
}

static StepKernel pick(int K, bool compact, int dry, bool bern, bool eq3, bool zlev, bool zpair = false, bool bin = false)
{
    if (bin) {
        if (zpair) return K == 1 ? pick_zp<1, true, true>(dry) : pick_zp<2, true, true>(dry);
        return K == 1 ? pick_zp<1, false, true>(dry) : pick_zp<2, false, true>(dry);
    }
    if (zpair) return K == 1 ? pick_zp<1, true, false>(dry) : pick_zp<2, true, false>(dry);
    if (K == 1) return bern ? pick_kb<1, true>(compact, dry, eq3, zlev) : pick_kb<1, false>(compact, dry, eq3, zlev);
    return bern ? pick_kb<2, true>(compact, dry, eq3, zlev) : pick_kb<2, false>(compact, dry, eq3, zlev);
}

cudaError_t launch_step(const StepArgs &a, int K, bool compact, int blocks, cudaStream_t st)
{
    // (lpm_api.cu asks for the binning epilogue - bin_cnt != null - only with the physics it is instantiated for)
    pick(K, compact, a.dry_mode, a.bern != 0, a.eq3 != 0, a.mg.nlev != 0 || a.drift != 0, a.zpair != 0, a.bin_cnt != nullptr)<<<blocks, kStepThreads, 0, st>>>(a);
    return cudaGetLastError();
}

int step_max_blocks_per_sm(int K, bool compact, int dry, bool bern, bool eq3, bool zlev, bool zpair)
{
    int nb = 0;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, pick(K, compact, dry, bern, eq3, zlev, zpair), kStepThreads, 0);
    return nb;
}

// a0: interleave the two snapshots of the current met interval into the pair buffer and turn the
// layout z-fastest: pair[(j*nx + i)*nz + k] = (F_s, F_s+1)(k, j, i).  A particle's z-cell changes
// every few steps (sigma_z per step ~ dz/3) while its column changes slowly, so with columns
// contiguous the 32 lanes of a column-sorted warp touch <= 8 128-byte lines per gather instead of
// one line per lane.  One thread per output texel: coalesced 32-byte writes, strided 16-byte reads
// (once per met interval, < 1 ms).
__global__ void __launch_bounds__(256) pair_repack_kernel(const float4 *__restrict__ s0, const float4 *__restrict__ s1,
                                                          Texel2 *__restrict__ pair, uint32_t nx, uint32_t ny, uint32_t nz,
                                                          uint32_t *__restrict__ uvmax)
{
    const uint64_t cells = (uint64_t)nx * ny * nz, plane = (uint64_t)nx * ny;
    float um = 0.f, vm = 0.f;  // largest |u|, |v| of the interval: bounds the advection of the plume box
    for (uint64_t o = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; o < cells; o += (uint64_t)gridDim.x * blockDim.x) {
        const uint64_t col = o / nz;
        const uint32_t k = (uint32_t)(o - col * nz);
        const uint64_t src = (uint64_t)k * plane + col;
        Texel2 t;
        t.a = __ldg(s0 + src);
        t.b = __ldg(s1 + src);
        pair[o] = t;
        um = fmaxf(um, fmaxf(fabsf(t.a.x), fabsf(t.b.x)));
        vm = fmaxf(vm, fmaxf(fabsf(t.a.y), fabsf(t.b.y)));
    }
    if (uvmax) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            um = fmaxf(um, __shfl_xor_sync(0xffffffffu, um, o));
            vm = fmaxf(vm, __shfl_xor_sync(0xffffffffu, vm, o));
        }
        if ((threadIdx.x & 31) == 0) {
            atomicMax(uvmax, __float_as_uint(um));   // non-negative floats order like their bit patterns
            atomicMax(uvmax + 1, __float_as_uint(vm));
        }
    }
}

cudaError_t launch_pair_repack(const float4 *s0, const float4 *s1, void *pair, int nx, int ny, int nz, uint32_t *uvmax, cudaStream_t st)
{
    if (uvmax) {
        const cudaError_t e = cudaMemsetAsync(uvmax, 0, 8, st);
        if (e != cudaSuccess) return e;
    }
    const uint64_t want = ((uint64_t)nx * ny * nz + 255) / 256;
    pair_repack_kernel<<<(int)(want < sm_count() * 8 ? want : sm_count() * 8), 256, 0, st>>>(s0, s1, (Texel2 *)pair, (uint32_t)nx, (uint32_t)ny, (uint32_t)nz,
                                                                                uvmax);
    return cudaGetLastError();
}

// a0, one snapshot (nt = 1): z-fastest copy of the caller's x-fastest snapshot
__global__ void __launch_bounds__(256) transpose_kernel(const float4 *__restrict__ s0, float4 *__restrict__ out, uint32_t nx, uint32_t ny,
                                                        uint32_t nz)
{
    const uint64_t cells = (uint64_t)nx * ny * nz, plane = (uint64_t)nx * ny;
    for (uint64_t o = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; o < cells; o += (uint64_t)gridDim.x * blockDim.x) {
        const uint64_t col = o / nz;
        out[o] = __ldg(s0 + (uint64_t)(uint32_t)(o - col * nz) * plane + col);
    }
}

cudaError_t launch_transpose(const float4 *s0, float4 *out, int nx, int ny, int nz, cudaStream_t st)
{
    const uint64_t want = ((uint64_t)nx * ny * nz + 255) / 256;
    transpose_kernel<<<(int)(want < sm_count() * 8 ? want : sm_count() * 8), 256, 0, st>>>(s0, out, (uint32_t)nx, (uint32_t)ny, (uint32_t)nz);
    return cudaGetLastError();
}

// a0, time weighting (R4; "interpolating ... in ... time"): for each of the m fused steps of
// the coming launch, out[s][o] = F_s + a_s (F_s+1 - F_s), texel by texel.  Interpolation in space and
// in time are both linear, so blending the texels first and sampling the blended field is the same
// function as sampling both snapshots and blending the samples; it halves the bytes the step kernel
// gathers (the L1 data pipe, not HBM or the ALUs, is what bounds that kernel) and its FMA count.
// Streaming: reads the pair buffer once, writes m x 16 bytes per cell.
struct BlendArgs {
    const Texel2 *pair;
    float4 *out;
    uint64_t cells;
    int32_t m;
    float a[kBlendDepth];
    BlendBox box;
    int32_t zpair;   // write z-pair texels {F(k), F(k+1)} (32 B) instead of F(k) (16 B)
};

// Only the columns a particle can reach are blended: a tile of 8 x 8 met columns is processed if a
// tile flagged by the step kernel (a particle sat there at the end of the previous launch) or a
// source column lies within the largest possible displacement of the coming steps,
// (|u|max dt + 5.768 sigma_h) per step (trilinear values are convex combinations of texels,
// |N(0,1)| <= 5.768 by R3), + 2 columns for the stencil, measured in whole tiles (rounded up).
__global__ void __launch_bounds__(256) blend_kernel(const __grid_constant__ BlendArgs B)
{
    const int nx = B.box.nx, ny = B.box.ny, ntx = (nx + kMaskTile - 1) / kMaskTile, nty = (ny + kMaskTile - 1) / kMaskTile;
    int mtx = 0, mty = 0;
    bool all = B.box.flags == nullptr;
    if (!all) {
        const float um = __uint_as_float(B.box.uvmax[0]), vm = __uint_as_float(B.box.uvmax[1]);
        const int mx = (int)ceilf(um * B.box.reach_x + B.box.walk_x) + 2, my = (int)ceilf(vm * B.box.reach_y + B.box.walk_y) + 2;
        mtx = (mx + kMaskTile - 1) / kMaskTile;
        mty = (my + kMaskTile - 1) / kMaskTile;
        if ((2 * mtx + 1) * (2 * mty + 1) > 1024) all = true;   // reach of the order of the domain: no point in masking
    }
    const uint32_t nz = (uint32_t)B.box.nz;
    constexpr int kParts = 4;   // blocks per tile (rows jj = part, part + kParts, ...): enough CTAs on small grids
    for (int item = blockIdx.x; item < ntx * nty * kParts; item += gridDim.x) {
        const int tile = item / kParts, part = item % kParts;
        const int ti = tile % ntx, tj = tile / ntx;
        if (!all) {
            int hit = 0;
            const int w = 2 * mtx + 1, nn = w * (2 * mty + 1);
            for (int t = threadIdx.x; t < nn; t += blockDim.x) {
                const int a = ti + t % w - mtx, b = tj + t / w - mty;
                if (a >= 0 && a < ntx && b >= 0 && b < nty && B.box.flags[b * ntx + a]) hit = 1;
            }
            if (threadIdx.x < B.box.n_src) {
                const int a = B.box.src_i[threadIdx.x] / kMaskTile, b = B.box.src_j[threadIdx.x] / kMaskTile;
                if (abs(a - ti) <= mtx && abs(b - tj) <= mty) hit = 1;
            }
            if (!__syncthreads_or(hit)) continue;
        }
        const uint32_t i0 = (uint32_t)(ti * kMaskTile), j0 = (uint32_t)(tj * kMaskTile);
        const uint32_t w = min((uint32_t)kMaskTile, (uint32_t)nx - i0), h = min((uint32_t)kMaskTile, (uint32_t)ny - j0);
        const uint32_t row = w * nz;   // the w columns of a tile row are contiguous (z fastest, then x)
        for (uint32_t jj = (uint32_t)part; jj < h; jj += kParts)
        for (uint32_t r = threadIdx.x; r < row; r += blockDim.x) {
            const uint64_t o = ((uint64_t)(j0 + jj) * (uint32_t)nx + i0) * nz + r;
            Texel2 tx;
            asm("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                : "=f"(tx.a.x), "=f"(tx.a.y), "=f"(tx.a.z), "=f"(tx.a.w), "=f"(tx.b.x), "=f"(tx.b.y), "=f"(tx.b.z), "=f"(tx.b.w)
                : "l"(B.pair + o));
            if (!B.zpair) {
#pragma unroll 4
                for (int s = 0; s < B.m; ++s) B.out[(uint64_t)s * B.cells + o] = lerp4(tx.a, tx.b, B.a[s]);
            } else {
                Texel2 ty;  // the next level of the same column (the top level pairs with itself)
                const uint64_t o1 = (r % nz) + 1u < nz ? o + 1 : o;
                asm("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                    : "=f"(ty.a.x), "=f"(ty.a.y), "=f"(ty.a.z), "=f"(ty.a.w), "=f"(ty.b.x), "=f"(ty.b.y), "=f"(ty.b.z), "=f"(ty.b.w)
                    : "l"(B.pair + o1));
#pragma unroll 4
                for (int s = 0; s < B.m; ++s) {
                    TexelZ w;
                    w.lo = lerp4(tx.a, tx.b, B.a[s]);
                    w.hi = lerp4(ty.a, ty.b, B.a[s]);
                    ((TexelZ *)B.out)[(uint64_t)s * B.cells + o] = w;
                }
            }
        }
    }
}

cudaError_t launch_blend(const void *pair, float4 *out, uint64_t cells, int m, const float *a, const BlendBox *box, bool zpair, cudaStream_t st)
{
    BlendArgs B;
    B.zpair = zpair ? 1 : 0;
    B.pair = (const Texel2 *)pair; B.out = out; B.cells = cells; B.m = m;
    for (int s = 0; s < kBlendDepth; ++s) B.a[s] = s < m ? a[s] : 0.0f;
    B.box = *box;
    const int tiles = ((box->nx + kMaskTile - 1) / kMaskTile) * ((box->ny + kMaskTile - 1) / kMaskTile);
    blend_kernel<<<tiles * 4 < sm_count() * 8 ? tiles * 4 : sm_count() * 8, 256, 0, st>>>(B);
    return cudaGetLastError();
}

// a0 for the 2-D fields of R12: out[s][c] = F_s + a_s (F_s+1 - F_s), x-fastest as the caller's arrays
struct SurfArgs {
    const float4 *s0, *s1;
    float4 *out;
    uint64_t cells2;
    int32_t m;
    float a[kBlendDepth];
};

__global__ void __launch_bounds__(256) blend_surface_kernel(const __grid_constant__ SurfArgs B)
{
    for (uint64_t c = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; c < B.cells2; c += (uint64_t)gridDim.x * blockDim.x) {
        const float4 f0 = __ldg(B.s0 + c), f1 = __ldg(B.s1 + c);
        for (int s = 0; s < B.m; ++s) B.out[(uint64_t)s * B.cells2 + c] = lerp4(f0, f1, B.a[s]);
    }
}

cudaError_t launch_blend_surface(const float4 *s0, const float4 *s1, float4 *out, uint64_t cells2, int m, const float *a, cudaStream_t st)
{
    SurfArgs B;
    B.s0 = s0; B.s1 = s1; B.out = out; B.cells2 = cells2; B.m = m;
    for (int s = 0; s < kBlendDepth; ++s) B.a[s] = s < m ? a[s] : 0.0f;
    const uint64_t want = (cells2 + 255) / 256;
    blend_surface_kernel<<<(int)(want < sm_count() * 8 ? (want ? want : 1) : sm_count() * 8), 256, 0, st>>>(B);
    return cudaGetLastError();
}

cudaError_t launch_inject(const InjectArgs &a, cudaStream_t st)
{
    uint64_t mx = 0;
    for (int r = 0; r < a.n_spec; ++r) mx = a.spec[r].count > mx ? a.spec[r].count : mx;
    int blocks = (int)((mx + 255) / 256);
    if (blocks < 1) blocks = 1;
    if (blocks > sm_count() * 8) blocks = sm_count() * 8;
    inject_kernel<<<blocks, 256, 0, st>>>(a);
    return cudaGetLastError();
}

}  // namespace lpm
