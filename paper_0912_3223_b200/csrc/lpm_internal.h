// lpm_internal.h — structs shared by the kernels (lpm_step.cu, lpm_bin.cu) and the host API
// (lpm_api.cu).  Not part of the public boundary (include/lpm.h).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/lpm.h"

// kernel formulation switches (round 2; all on: measured one by one on c4, profiles/r02_*): packed FFMA2 arithmetic,
// MUFU.SQRT, 32-bit texel indices, direct-mapped deposit window
#ifndef LPM_FUSED_LONG
#define LPM_FUSED_LONG 64
#endif

namespace lpm {

constexpr int kMaxFused = 16;        // model steps fused into one launch (table lives in kernel params)
constexpr int kMaxFusedLong = LPM_FUSED_LONG;    // ... when every step samples the same met buffer (one snapshot) and nothing goes through the
                                     // deposit tables (their fixed-point sums hold 256 x 16 increments): small, launch-latency-bound
                                     // runs like c1 ("fewer particles ... GPU spends most of the time on initialization")
constexpr int kBlendDepth = kMaxFused;  // time-blended met buffers kept: one per fused step
constexpr int kMaxLevels = 64;       // non-uniform vertical met levels held in the kernel parameters
constexpr int kSortPeriod = 32;      // least number of model steps between two gather-locality sorts of a release (auto: 32..64)
constexpr int kStepThreads = 256;    // CTA size of the step kernel
constexpr int kScanTile = 4 * kStepThreads;  // particles per look-back tile (compaction): 4 per thread

// Per-step scalars, host-computed in double (DESIGN.md §3 R4, R8).
struct StepEntry {
    double G[LPM_MAX_NUCLIDES];  // G_k(t_n): activity = q * G (decay and uniform dry loss folded in)
    float Gf[LPM_MAX_NUCLIDES];  // (float)G_k(t_n), the factor the per-step fp32 arithmetic uses
    float Gp[LPM_MAX_NUCLIDES];  // (float)(G_k(t_n) * p_dry,k): uniform dry deposit of one step per unit q
    float Gps[LPM_MAX_NUCLIDES]; // Gp * S_dry,k: the same in the fixed-point units of the deposit tables
    // deposit increments per unit activity in table units: p * S * Er, with Er = exp(lambda_k (t_n - t_launch)) when the
    // map decays on the ground (R13: it is kept referred to a fixed time, so later increments weigh more), else 1
    float Pd[LPM_MAX_NUCLIDES], Pw[LPM_MAX_NUCLIDES];
    float Oid[LPM_MAX_NUCLIDES], Oiw[LPM_MAX_NUCLIDES];  // 1 / (S * Er): table units back to activity (off-map ledger)
    double Eg[LPM_MAX_NUCLIDES];                         // exp(lambda_k (t_n - t_ref)): direct deposits (Bernoulli form)
    float a;                     // time weight between snapshot `snap` and `snap + 1`
    int32_t snap;                // bits 0..15 snapshot index, bit 16 = raining
    uint32_t buf;                // which time-blended met buffer holds F(t_n) (a0)
    uint32_t pad_;
};

struct GridF {  // fp32 view of a grid, exactly as the kernels use it
    int32_t nx, ny, nz;
    float x0, y0, z0;          // (float) lower corner
    float inv_dx, inv_dy, inv_dz;  // (float)(1.0 / d)
    // derived, for the met sampling R4: the upper clamp of the grid coordinate, the largest lower
    // corner index, and the element strides to the upper corner (0 on an axis with a single cell:
    // i1 = min(i0 + 1, n - 1) = i0 + 1 whenever n >= 2, because i0 <= n - 2)
    float cx, cy, cz;          // (float)(-p0/d - 1/2): grid coordinate of the stencil g = p * inv_d + c
    float fx1, fy1, fz1;       // (float)(n - 1)
    int32_t ix2, iy2, iz2;     // max(n - 2, 0)
    uint32_t ex, ey, ez;       // element strides of cell (i, j, k) in the sampled buffer: z-fastest (nz, nx*nz, 1)
                               // for the library's met buffers (x-fastest (1, nx, nx*ny) is the caller's layout)
    uint32_t sx, sy, sz;       // stride to the upper corner on each axis: n > 1 ? e : 0
    int32_t nlev;              // 0: uniform vertical levels; else nz non-uniform level heights, ascending
    float zlev[kMaxLevels];
};

enum DryMode : int32_t { kDryNone = 0, kDryUniform = 1, kDryLayer = 2 };

struct StepArgs {
    // particle store
    float4 *xyzq;
    float *q1;
    uint32_t *pid;        // compact mode only
    // meteorology (a0): `blend` = the library's z-fastest float4 buffers [n_buf][cells]; buffer
    // tab[s].buf holds the field at the time of fused step s, F(t_n) = F_s + a (F_s+1 - F_s)
    const float4 *blend;
    const float4 *surf;   // kz_mode 1 (R12): time-blended 2-D fields (u*, 1/L, Hz, -) [n_buf][ny][nx], x fastest; else null
    uint64_t snap_cells;  // cells per snapshot
    GridF mg;
    float bx0, bx1, by0, by1;  // lateral boundary (met box), fp32
    // deposition map
    GridF cg;
    double *dep;          // [K][ny][nx]
    uint64_t dep_stride;
    float dep_scale[2 * LPM_MAX_NUCLIDES];       // fixed-point scales of the CTA-private deposit sums (powers of two): [2k] dry, [2k+1] wet
    double dep_inv_scale[2 * LPM_MAX_NUCLIDES];  // their inverses
    int32_t zpair, keys_by_slot;             // the blended buffers hold z-pair texels (32 B: both z corners), B8; fused sort keys indexed by slot, not by list position
    int32_t eq3, drift;                      // kz_mode 1: Kz from Eq.(3) per particle; drift: + dKz/dz dt (departure from the paper)
    int32_t any_dep, bern;                   // some sink deposits through the tables; dep_mode 1: Bernoulli deposition (R11)
    // a8 fused: non-null when this launch ends on a binning step: count grid, sum grids [K][cells3], fixed-point scales
    uint32_t *bin_cnt;
    double *bin_conc;
    uint64_t bin_cells3;
    float bin_scale[LPM_MAX_NUCLIDES];
    double bin_inv_scale[LPM_MAX_NUCLIDES];
    // physics
    float dt, sigma_h, kz_min, H, h_dep;
    int32_t dry_mode, absorb;
    float p_dry[LPM_MAX_NUCLIDES], p_wet[LPM_MAX_NUCLIDES];
    float rx0, rx1, ry0, ry1;
    uint32_t seed_lo, seed_hi;
    uint32_t rk[20];      // Philox round keys (k0, k1) of rounds 0..9: key + r * Weyl constants (R1)
    // ledger: double [K][8]: 2 dry, 3 wet, 4 decayed, 5 exited, 6 offgrid
    double *ledger;
    double dec_scale[LPM_MAX_NUCLIDES];  // (1 - f_lambda) * (1 - p_dry if uniform)
    double wet_scale[LPM_MAX_NUCLIDES];  // (1 - p_dry if uniform) * p_wet
    float wet_scale_f[LPM_MAX_NUCLIDES]; // (float)wet_scale
    // population (slot-addressed mode): slots [0, n) of the release block starting at `base`
    uint64_t base, n, n_prev;  // slots >= n_prev are born inside this launch
    const uint32_t *perm;      // gather-locality pass: slots [0, n_perm) listed in dual-cell order, or null
    uint64_t n_perm;           // slots [n_perm, n) are walked in slot order
    const uint64_t *n_live;    // device: length of the live part of `perm` (particles that had left the domain at the
                               // sort are not listed); the kernel walks the positions [0, min(*n_live, n_perm))
    uint8_t *mask;             // non-null: flag the mask tile of each particle's met column at the end of the launch
    int32_t mask_ntx, pad2_;
    uint32_t *keys_out, *hist_out;  // non-null: the launch before a sort leaves each slot's dual-cell key and the histogram
    uint32_t n_keys, pad1_;
    uint64_t pid_offset, pid_stride;
    uint64_t rel_N, rel_c;     // count mode: N (global count); rate mode: c slots per step
    int64_t rel_s_start, rel_S;
    double emit[LPM_MAX_NUCLIDES];  // activity per particle at birth
    float sx, sy, sz;               // source point
    // compact mode: device-side control block
    uint64_t *ctrl;      // [0] n_active, [1] ticket, [2] n_out
    uint64_t *tile_state;
    uint32_t *holes;     // compact + unordered store: slots of the particles that left in this step (count in ctrl[4]); null = stable scan
    // time
    uint64_t step0;
    int32_t m_steps;
    StepEntry tab[kMaxFusedLong];
};

// compact mode: newborn particles of one step, appended behind the live ones
struct InjectSpec {
    uint64_t first_pid, count, pid_stride;
    int32_t rel_index, pad_;
    float sx, sy, sz;
    float q[LPM_MAX_NUCLIDES];   // (float)(emit_k / G_k(t_n))
};
struct InjectArgs {
    float4 *xyzq;
    float *q1;
    uint32_t *pid;
    uint64_t *ctrl;       // [0] n_in, [1] ticket, [2] n_out of the previous step
    uint64_t *log_slot;   // injected count of this step (may be null)
    uint64_t capacity;
    int32_t n_spec, K;
    InjectSpec spec[LPM_MAX_RELEASES];
};

struct BinArgs {
    const float4 *xyzq;
    const float *q1;
    uint64_t n;               // slots to bin (slot-addressed mode)
    const uint64_t *n_dev;    // compact mode: read n from here
    GridF cg;
    uint32_t *cnt;
    double *conc;             // [K][cells3] sums of q
    uint64_t cells3;
    int32_t K, pad_;
    // fixed-point scale of the CTA-private sums (power of two; 2^19 <= q_max * scale < 2^20) and its inverse
    float scale[LPM_MAX_NUCLIDES];
    double inv_scale[LPM_MAX_NUCLIDES];
    uint64_t *n_binned;       // device counter: += particles binned (active and inside the grid)
};

// launchers implemented in the .cu files; all return the cudaError of the launch
cudaError_t launch_step(const StepArgs &a, int K, bool compact, int grid_blocks, cudaStream_t st);
int step_max_blocks_per_sm(int K, bool compact, int dry_mode, bool bern, bool eq3, bool zlev, bool zpair);
cudaError_t launch_inject(const InjectArgs &a, cudaStream_t st);
cudaError_t launch_sort_by_cell(const float4 *xyzq, uint64_t n, GridF g, uint32_t *keys, uint32_t *hist, uint32_t *partial,
                                uint32_t *perm, uint64_t *live_out, cudaStream_t st);
cudaError_t launch_sort_finish(const uint32_t *keys, uint64_t n, uint32_t n_keys, uint32_t *hist, uint32_t *partial, const uint32_t *list_old,
                               uint64_t n_old, const uint64_t *live_old, uint32_t *perm, uint64_t *live_out, cudaStream_t st);
cudaError_t launch_fill_holes(float4 *xyzq, float *q1, uint32_t *pid, uint64_t *ctrl, const uint32_t *holes, uint32_t *src, uint32_t *dst,
                              cudaStream_t st);
cudaError_t launch_sort_records(float4 *xyzq, float *q1, uint32_t *pid, const uint64_t *n_dev, uint64_t capacity, GridF g, uint32_t *keys,
                                uint32_t *hist, uint32_t *partial, float4 *xyzq_alt, float *q1_alt, uint32_t *pid_alt, cudaStream_t st);
uint64_t sort_partial_entries(uint64_t n_cells);
cudaError_t run_probe(int kind, uint64_t footprint_bytes, void *scratch_dev, uint64_t scratch_bytes, int reps, double *ops,
                      cudaStream_t st);
cudaError_t launch_pair_repack(const float4 *s0, const float4 *s1, void *pair, int nx, int ny, int nz, uint32_t *uvmax, cudaStream_t st);
cudaError_t launch_blend_surface(const float4 *s0, const float4 *s1, float4 *out, uint64_t cells2, int m, const float *a, cudaStream_t st);
cudaError_t launch_transpose(const float4 *s0, float4 *out, int nx, int ny, int nz, cudaStream_t st);
// plume mask (a0): blend only the met columns a particle can reach during the coming launch.  The met
// columns are grouped in tiles of kMaskTile x kMaskTile; the step kernel flags the tiles that hold a
// particle, the blend kernel processes a tile if a flagged tile (or a source) lies within reach.
constexpr int kMaskTile = 8;
struct BlendBox {
    const uint8_t *flags;   // device: one byte per tile [nty][ntx], != 0 = holds a particle; null = whole field
    const uint32_t *uvmax;  // device: {|u|max, |v|max} of the current met interval, float bits
    int32_t nx, ny, nz;
    float reach_x, reach_y;    // columns per (m/s) of wind:  steps * dt / dx
    float walk_x, walk_y;      // columns of random walk: steps * 5.768 sigma_h / dx  (|N(0,1)| <= sqrt(48 ln 2) by construction, R3)
    int32_t n_src;
    int32_t src_i[LPM_MAX_RELEASES], src_j[LPM_MAX_RELEASES];   // source columns (newborn particles)
};
cudaError_t launch_blend(const void *pair, float4 *out, uint64_t cells, int m, const float *a, const BlendBox *box, bool zpair, cudaStream_t st);
cudaError_t launch_bin(const BinArgs &a, int blocks, cudaStream_t st);
cudaError_t launch_conc_readout(const double *conc, float *out, uint64_t cells3, int K, const double *scale, cudaStream_t st);
cudaError_t launch_dose_accum(const double *conc, double *dose, uint64_t cells3, int K, const double *scale, cudaStream_t st);
cudaError_t launch_dep_readout(const double *dep, float *out_f32, double *out_f64, uint64_t cells2, int K, const double *scale, cudaStream_t st);
cudaError_t launch_dep_rebase(double *dep, uint64_t cells2, double factor, cudaStream_t st);
cudaError_t launch_airborne(const float4 *xyzq, const float *q1, uint64_t n, const uint64_t *n_dev, int K, double *out2, cudaStream_t st);
cudaError_t launch_export(const float4 *xyzq, const float *q1, uint64_t n, const uint64_t *n_dev, float4 *out, uint8_t *status, cudaStream_t st);
cudaError_t launch_import(float4 *xyzq, uint64_t n, const uint8_t *status, cudaStream_t st);
cudaError_t launch_iota(uint32_t *pid, uint64_t n, uint64_t offset, uint64_t stride, cudaStream_t st);
cudaError_t launch_check_affine(const uint32_t *pid, uint64_t n, uint64_t offset, uint64_t stride, uint32_t *bad, cudaStream_t st);
cudaError_t launch_count_nonzero(const uint32_t *cnt, uint64_t cells3, uint64_t *out, cudaStream_t st);
int sm_count();   // SMs of the current device (cached)
cudaError_t launch_qmax(const float4 *xyzq, const float *q1, uint64_t n, int K, float *out2, cudaStream_t st);
cudaError_t launch_test_philox(uint64_t seed, uint64_t step, uint32_t stream, uint64_t pid0, uint64_t n, uint32_t *out, cudaStream_t st);
cudaError_t launch_test_curand_philox(uint64_t seed, uint64_t step, uint64_t pid0, uint64_t n, uint32_t *out, cudaStream_t st);
cudaError_t launch_test_box_muller(const uint32_t *r, uint64_t n, float *out, cudaStream_t st);
cudaError_t launch_test_normals(uint64_t seed, uint64_t step, uint64_t pid0, uint64_t n, float *out, cudaStream_t st);
cudaError_t launch_test_sample(const float4 *blend, GridF mg, float kz_min, const float4 *xyz, uint64_t n, float4 *out,
                               cudaStream_t st);

}  // namespace lpm
