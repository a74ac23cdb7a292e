/* lpm.h — C ABI of the B200-native Lagrangian particle step + binning library.
 *
 * The hot path of arxiv/paper_0912_3223 (Molnar, Szakaly, Meszaros, Lagzi: "Air pollution
 * modelling using a Graphics Processing Unit with CUDA"), cited below as P:Lnn = PAPER.md line nn:
 * point source releasing particles with assigned activity every time step, each step per
 * particle = linear sampling of gridded weather in x, y, z and time -> turbulent diffusion
 * coefficient -> move by wind -> move by turbulent diffusion -> dry / wet deposition test ->
 * inactive at the boundary (Eq.(1)(2)), radioactive decay from the half-life
 * (P:L84), and the summation of particle activity on a rectangular grid every n-th step.
 * Readings of everything the paper leaves open: DESIGN.md §3 (R1..R10).
 *
 * Conventions
 *  - Every function returns int32_t: LPM_OK (0) or a negative lpm_status.  No exceptions, no C++
 *    types, no torch types cross this boundary.
 *  - Pointers named *_dev are DEVICE pointers (cudaMalloc / torch CUDA tensors); *_host are host
 *    pointers; small structs are host structs copied at the call.
 *  - OWNERSHIP: the caller owns every device buffer (workspace, met snapshots, outputs).  The
 *    library borrows `workspace_dev` and `meteo.fields_dev` for the life of the handle and never
 *    frees caller memory.  The library keeps re-packed, time-blended copies of the two snapshots of
 *    the current met interval: snapshot data must be in place before the first step of the interval
 *    that uses it, and later changes must go through lpm_upload_meteo (which invalidates the copies).
 *  - One handle = one GPU = one CUDA stream.  Calls enqueue work on that stream and return; calls
 *    that return host scalars (lpm_num_active, lpm_ledger, lpm_get_particles' count) synchronise
 *    the stream first.  A handle is not thread-safe.
 *  - There is NO CPU fallback: without an sm_100 device lpm_create returns LPM_ERR_NO_DEVICE.
 *  - Units: SI (m, s, Bq).  Grids are x-fastest: index = (k*ny + j)*nx + i.
 */
#ifndef LPM_H_
#define LPM_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define LPM_MAX_NUCLIDES 2
#define LPM_LEDGER_FIELDS 7 /* emitted, airborne, dry, wet, decayed, exited, dep_offgrid */
#define LPM_MAX_RELEASES 8

typedef enum {
    LPM_OK = 0,
    LPM_ERR_INVALID_ARG = -1,
    LPM_ERR_NO_DEVICE = -2,          /* no sm_100 CUDA device; there is no CPU fallback       */
    LPM_ERR_WORKSPACE_TOO_SMALL = -3,
    LPM_ERR_CAPACITY = -4,           /* a release does not fit into params.capacity           */
    LPM_ERR_STATE = -5,              /* call order (e.g. release registered after its start)  */
    LPM_ERR_CUDA = -6                /* sticky; text via lpm_last_error                       */
} lpm_status;

typedef enum { LPM_BOUNDARY_OPEN = 0, LPM_BOUNDARY_ABSORB = 1 } lpm_boundary_mode;
typedef enum { LPM_DEP_EXPECTED = 0, LPM_DEP_BERNOULLI = 1 } lpm_dep_mode;

/* Regular grid of nx*ny*nz cells of size dx*dy*dz with lower corner (x0, y0, z0). */
typedef struct {
    int32_t nx, ny, nz, reserved;
    double x0, y0, z0, dx, dy, dz;
} lpm_grid;

/* Meteorology: nt snapshots at t0 + s*dt_snap, each nz*ny*nx cell-centred texels
 * float4 = (u, v, w, Kz) [m/s, m/s, m/s, m^2/s], layout [nt][nz][ny][nx], x fastest, 16-byte
 * aligned.  Sampling is trilinear in space, linear in time, edge-clamped (R4).  Kh: constant
 * horizontal diffusivity.  H_mix: reflecting lid (R6).  kz_min: floor on the sampled Kz. */
typedef struct {
    lpm_grid grid;
    int32_t nt;
    int32_t kz_mode;          /* 0: Kz is the w component of the texels (sampled like the wind); 1: Kz from Eq.(3)
                               * per particle with the 2-D fields of surface_dev (R12)       */
    double t0, dt_snap;
    const void *fields_dev;
    double Kh, H_mix, kz_min;
    const void *surface_dev;  /* kz_mode 1: float4 (u* [m/s], 1/L [1/m], Hz [m], unused) [nt][ny][nx], x fastest,
                               * 16-byte aligned, borrowed like fields_dev; else ignored (may be NULL)             */
    const double *z_levels_host; /* NULL: uniform vertical levels z0 + (k + 1/2) dz.  Else HOST array of grid.nz
                               * strictly ascending level heights [m] ("vertical weather information is
                               * nonlinear"; nz <= 64): linear between the bracketing levels, clamped outside;
                               * copied (as fp32) by lpm_create                                                    */
} lpm_meteo;

/* Isotope constants. half_life_s <= 0 means stable. */
typedef struct {
    double half_life_s;
    double vd;         /* dry deposition velocity, m/s  */
    double lambda_wet; /* wet scavenging coefficient, 1/s */
} lpm_nuclide;

typedef struct {
    double dt;              /* time step, s (10 s)                                       */
    uint64_t seed;          /* Philox key (R1)                                                  */
    uint64_t capacity;      /* maximum number of particle slots                        */
    int32_t boundary_mode;  /* lpm_boundary_mode; the boundary is the met-grid box (R7)         */
    int32_t compact;        /* 1: stream compaction of exited particles after every step.  Stable (survivors keep
                             * their order = id order) when gather_sort is off; with gather_sort on the store
                             * is unordered (re-sorted by met cell) and holes are filled from the tail */
    double h_dep;           /* dry deposition acts where z' < h_dep; h_dep >= H_mix: everywhere */
    int32_t bin_every;      /* concentration binning cadence in steps ("n"); 0 = never   */
    int32_t steps_per_launch; /* 0 = auto (16; 64 with a single met snapshot and no deposition: small runs are
                               * launch-latency-bound); 1 = one model step per kernel launch; m > 1 fuses up to
                               * min(m, 16 or 64) steps per launch with the particle state in registers */
    int32_t gather_sort;      /* gather-locality pass (slots listed in the order of the lower-corner met
                               * cell of their trilinear stencil): 0 = auto (from 65536 particles, every
                               * 32 to 64 steps: about the time the horizontal walk needs to cross a met
                               * cell), p > 0 = always, every p model steps (1 = before every launch),
                               * -1 = never.  Results per particle do not depend on it.  With compact = 1
                               * the records themselves are sorted (the id travels with the particle), so
                               * the store is then in met-cell order, not in id order.             */
    int32_t dose;             /* 1: accumulate the time-integrated concentration (Fig. 2b "time
                               * integrated dosage") at every cadence binning; read with lpm_dose        */
    int32_t dep_mode;         /* lpm_dep_mode: 0 expected-mass deposition (every step removes the fraction p
                               * of the activity), 1 the paper's stochastic form: one
                               * Bernoulli trial per nuclide and sink per step from Philox stream 1, an
                               * event deposits the nuclide's whole activity once; a particle that
                               * carries nothing any more becomes inactive (status 2)                */
    int32_t drift;            /* 1: LABELLED DEPARTURE from the paper: z' also gets + dKz/dz * dt,
                               * the drift correction of the well-mixed random walk, with dKz/dz the z-slope of
                               * the sampled (gridded) Kz at X_old; 0 (default) is the paper's Eq.(1)(2).
                               * Not with kz_mode 1 (INVALID_ARG)                                    */
    int32_t texel_pairs;      /* layout of the time-blended met buffers the step kernel gathers from (B8):
                               * -1 = one 16-byte texel F(k) per met cell (8 gathers per step); 1 = 32-byte
                               * texels {F(k), F(k+1)}: 4 gathers per step, twice the bytes per blended cell;
                               * 0 = auto: pairs when capacity >= 16 x the met cells (the blending kernel's
                               * extra writes are then small beside the step kernel's gain).  Results are
                               * bit-identical either way.  Pairs need the default physics on the
                               * slot-addressed store: compact = 0, nt > 1, dep_mode 0, kz_mode 0, uniform
                               * levels, drift 0 (auto: 16-byte texels otherwise; 1: INVALID_ARG)     */
    int32_t ground_decay;     /* 1: what has been deposited keeps decaying on the ground with its nuclide's half-life
                               * (SURVEY 8(c) R8 "a read-out-time option", 8(f)3; R13): the increments of step n
                               * decay from t_n on, and lpm_deposition* return the map as it is at the current time.
                               * 0 (default): the map is the cumulative deposited activity, never decayed.  The ledger
                               * (what left the air) is the same either way                            */
} lpm_params;

typedef struct {
    double x, y, z;         /* source point ("single point source")                       */
    double t_start, t_end;  /* release interval; first step ceil(t_start/dt), over
                             * max(1, ceil((t_end - t_start)/dt)) steps (R9)                     */
} lpm_source;

typedef struct lpm_handle lpm_handle;

/* ---- host-only entry points (usable without a GPU) --------------------------------------- */

/* Library version: major*10000 + minor*100 + patch. */
int32_t lpm_version(void);

/* Static text for a status code. */
const char *lpm_status_string(int32_t status);

/* Bytes of device workspace lpm_create needs for params->capacity particle slots (the capacity travels inside
 * lpm_params, as for lpm_create, not as an argument of its own) (particle SoA store, grids, ledger, scan state,
 * read-out staging, the z-fastest time-blended met buffers (16 bytes per met cell and fused step) and,
 * when meteo->nt > 1, the interleaved snapshot-pair buffer of the current met interval: 32 bytes per
 * met cell).  Only the grid and nt of `meteo` are read.  Errors: INVALID_ARG (as lpm_create for the same arguments;
 * among them: a met grid of 2^28 cells or more with nt > 1 - the step kernel's 32-bit texel index spans all 16 blended
 * buffers - or of 2^31 or more cells at all). */
int32_t lpm_workspace_bytes(const lpm_grid *conc_grid, const lpm_meteo *meteo, const lpm_params *params,
                            int32_t n_nuclides, uint64_t *bytes_host);

/* R9 release schedule, count mode: how many of the LOCAL particles (global ids pid_offset +
 * l*pid_stride < n_particles) are born at steps <= step, for a release starting at step s_start
 * and lasting S steps: global particle j is born at s_start + floor(j*S/n_particles). */
int32_t lpm_schedule_born(uint64_t n_particles, uint64_t pid_offset, uint64_t pid_stride,
                          int64_t s_start, int64_t S, int64_t step, uint64_t *born_host);

/* ---- life cycle ---------------------------------------------------------------------------- */

/* Create a simulation.  `conc_grid` is the 3-D concentration grid; the 2-D deposition map is its
 * (x, y) footprint.  `cuda_stream` is a cudaStream_t (NULL = default stream).  The workspace is
 * zeroed (asynchronously).  Errors: INVALID_ARG (null pointers, n_nuclides not in 1..2,
 * non-positive sizes, misaligned buffers), NO_DEVICE, WORKSPACE_TOO_SMALL, CUDA. */
int32_t lpm_create(const lpm_grid *conc_grid, const lpm_meteo *meteo, const lpm_nuclide *nuclides,
                   int32_t n_nuclides, const lpm_params *params, void *workspace_dev,
                   uint64_t workspace_bytes, void *cuda_stream, lpm_handle **out);

int32_t lpm_destroy(lpm_handle *h);

/* Start the same run again from step 0 on the same handle: the registered releases, the rain box, the grids' geometry and
 * the meteorology stay; the step index, the output grids, the deposition map, the ledger, the injected log and every
 * cached list / blended met buffer are cleared (asynchronously; the particle store needs no clearing: a slot is
 * initialised when its particle is born).  The results of the second run equal those of the first.  The device-side unit
 * counters behind lpm_get_timing's [4] and [5] start again at 0 as well: after a restart they count from the restart, while
 * the times and launch counts keep accumulating since lpm_set_timing (call lpm_set_timing again for a clean slate).
 * Errors: STATE (the particle state was installed by lpm_set_particles: there is no release to start again), CUDA. */
int32_t lpm_restart(lpm_handle *h);

/* Axis-aligned rain box over the full column, active for t_start <= t_n < t_end, tested at the
 * start of the step ("wet deposition only occurs in case of precipitation"; G6). */
int32_t lpm_set_rain(lpm_handle *h, double x0, double x1, double y0, double y1, double t_start,
                     double t_end);

/* Register a release.  total_activity_host[k] is the activity of nuclide k
 * emitted over the whole release, split evenly over the particles.  Count mode (n_particles > 0):
 * particle j of n_particles is born at step s_start + floor(j*S/n_particles); only the ids
 * pid_offset + l*pid_stride are simulated (pid-strided subsample / multi-GPU shard), each still
 * carrying total/n_particles.  Rate mode (n_particles == 0): c = round(particles_per_s*dt) slots
 * per step, pid = pid_offset + (step - s_start)*c + j; when capacity is short the highest j are
 * skipped (never renumbered); pid_stride must be 1.  Particle ids must stay below 2^32.
 * Errors: CAPACITY, STATE (release starts before the current step), INVALID_ARG. */
int32_t lpm_release(lpm_handle *h, const lpm_source *src, const double *total_activity_host,
                    uint64_t n_particles, double particles_per_s, uint64_t pid_offset,
                    uint64_t pid_stride);

/* Advance n_steps model steps.  Every params.bin_every-th step the concentration
 * grid is re-binned from the particle state: on the slot-addressed store by the step launch that ends on that
 * step, while the particles are still in registers; on the compact store by the stand-alone binning kernel. */
int32_t lpm_step(lpm_handle *h, int32_t n_steps);

/* ---- outputs -------------------------------------------------------------------------------- */

/* Concentration in Bq m^-3, float [K][nz][ny][nx], of the particle state at the current step
 * (re-bins first if the internal grid is stale).  P:L108 "At the end of every n-th time step the activity of particles
 * is calculated ... Activities or masses of particles are summarized on a rectangular grid"; P:L136-138 (the fields on
 * a 3-D grid that the paper compares cell by cell). */
int32_t lpm_concentration(lpm_handle *h, float *out_dev);
/* Time-integrated concentration in Bq s m^-3, float [K][nz][ny][nx]: sum over the cadence binnings so far
 * of (concentration at that binning) x (bin_every * dt) (rectangle rule; needs params.dose = 1, else STATE). */
int32_t lpm_dose(lpm_handle *h, float *out_dev);
/* Particle counts per cell, uint32 [nz][ny][nx], same snapshot rule (the same summation with weight 1 per
 * active particle - the sample size behind each cell of the grid of P:L136). */
int32_t lpm_counts(lpm_handle *h, uint32_t *out_dev);
/* Deposited activity in Bq m^-2, float [K][ny][nx] ("finally testing for dry and wet depositions", P:L84-86
 * "remove from the atmosphere to the surface by dry and wet pathways"): cumulative and never decayed with params.ground_decay = 0 (default);
 * with ground_decay = 1 what lies on the ground keeps decaying and the map is returned as it is at the current time. */
int32_t lpm_deposition(lpm_handle *h, float *out_dev);
/* Same map at full precision, double [K][ny][nx] (the accumulator itself, scaled by 1/area). */
int32_t lpm_deposition_f64(lpm_handle *h, double *out_dev);

/* ---- test hooks / checkpoint ---------------------------------------------------------------- */

/* Re-bin the current particle state into the internal grids now. */
int32_t lpm_bin_now(lpm_handle *h);
/* Number of particle slots in use (born, minus compacted-out). Synchronises. */
int32_t lpm_num_active(lpm_handle *h, uint64_t *n_host);
int32_t lpm_step_index(lpm_handle *h, uint64_t *step_host);
/* The activity of a particle is q * scale[k]: q is the stored fp32 value, scale[k] =
 * G_k(t) the host-side fp64 decay (and uniform dry-deposition) factor at the current step (R8). */
int32_t lpm_mass_scale(lpm_handle *h, double *scale_host /* [K] */);
/* Copy out the particle state: xyzq_dev float4 (x, y, z, q0) per slot, q1_dev (K = 2, may be
 * NULL), pid_dev uint32 global particle ids (may be NULL; slot-addressed store: pid_offset + l * pid_stride for slot l
 * of a release block), status_dev uint8 0 = active, 1 = exited, 2 = deposited all it carried
 * (dep_mode 1) (may be NULL).
 * Buffers must hold capacity entries; *n_host receives the slot count.  Exited particles report
 * their exit position.  With several releases each release owns a block of slots that starts at a multiple of
 * 64; the unused slots between two blocks read as zeros (binning, ledger and deposition skip them). */
int32_t lpm_get_particles(lpm_handle *h, void *xyzq_dev, float *q1_dev, uint32_t *pid_dev,
                          uint8_t *status_dev, uint64_t *n_host);
/* Replace the particle state by n slots (all treated as already born; pid_dev NULL = 0..n-1;
 * status_dev NULL = all active) and set the step index.  Registered releases keep running only
 * in compact mode (append); in slot-addressed mode they are dropped.  With compact = 0 the id of a particle is
 * implied by its slot, so pid_dev (if given) must be affine, pid[l] = pid[0] + l * (pid[1] - pid[0]) with a positive
 * stride - exactly what lpm_get_particles reports for one release, strided or not - else INVALID_ARG: a run
 * restarted from lpm_get_particles' output continues bit for bit.  The output grids are kept; with
 * ground_decay = 1 the deposition map is first brought to the present and then regarded as the ground
 * activity at the new step index. */
int32_t lpm_set_particles(lpm_handle *h, const void *xyzq_dev, const float *q1_dev,
                          const uint32_t *pid_dev, const uint8_t *status_dev, uint64_t n,
                          uint64_t step_index);
/* Mass ledger, double [K][LPM_LEDGER_FIELDS]: emitted, airborne, dry, wet, decayed, exited,
 * dep_offgrid (the part of dry+wet that fell outside the map).  emitted = airborne + dry + wet +
 * decayed + exited up to fp32 rounding.  Synchronises. */
int32_t lpm_ledger(lpm_handle *h, double *out_host);
/* Particles injected at `step` (rate mode log; 0 if the step has not run). Synchronises. */
int32_t lpm_injected(lpm_handle *h, uint64_t step, uint64_t *n_host);
/* Text of the last error on this handle ("" if none).  Owned by the handle. */
const char *lpm_last_error(lpm_handle *h);
/* Number of kernel launches issued by this handle so far (bench.py's gpu_launches). */
int32_t lpm_launch_count(lpm_handle *h, uint64_t *n_host);
/* *on_host = 1 when this handle's blended met buffers hold 32-byte z-pair texels (lpm_params.texel_pairs, after the
 * auto rule), else 0 */
int32_t lpm_texel_pairs(lpm_handle *h, int32_t *on_host);

/* ---- host-buffer entry points (end-to-end use: weather arrives from, results go to, host memory) */

/* Copy n_snapshots meteorological snapshots from HOST memory (pinned for full PCIe speed) into
 * the borrowed device array meteo.fields_dev, starting at snapshot index `first` (P:L104-106:
 * the weather data of the coming interval are loaded before it is simulated).  Asynchronous on
 * the handle's stream.  Errors: INVALID_ARG (null, range outside [0, nt)), CUDA. */
int32_t lpm_upload_meteo(lpm_handle *h, int32_t first, int32_t n_snapshots, const void *fields_host);
/* lpm_concentration / lpm_deposition into HOST buffers: read-out kernel into a staging area of the
 * workspace, then a device-to-host copy on the handle's stream; returns after the copy has
 * completed (the stream is synchronised), so out_host is valid on return. */
int32_t lpm_concentration_host(lpm_handle *h, float *out_host);
int32_t lpm_deposition_host(lpm_handle *h, float *out_host);

/* ---- timing hooks (bench.py's per-kernel roofline numbers) --------------------------------- */

/* enable != 0: bracket every step-kernel and every binning-kernel launch of this handle with CUDA
 * events on the handle's stream (two cudaEventRecord per launch); also clears the totals. */
int32_t lpm_set_timing(lpm_handle *h, int32_t enable);
/* Synchronises, then returns out_host[0] = total ms in step kernels, [1] = their launch count,
 * [2] = total ms in binning kernels (the memset of the grids included), [3] = their launch count,
 * [4] = particle-steps EXECUTED (born and still active particles x steps; counted by the step kernels themselves, so
 *       particles that have left the domain or deposited everything do not count),
 * [5] = particles BINNED (active and inside the concentration grid; counted by the binning kernel),
 * [6] = total ms in gather-locality sort passes, [7] = their count,
 * [8] = born particles x steps of the timed step launches (host count of the release schedule R9: the same as [4]
 *       while no particle has become inactive; slot-addressed store only, 0 with compact = 1),
 * [9]  = total ms of the step launches that carried the fused binning epilogue (slot-addressed store: the launch that
 *        ends on a binning step bins its particles itself; these launches are also part of [0] and [1]),
 * [10] = their count, [11] = total ms of the step launches directly before them (same population to within 16 steps
 *        of births); [12] = born particles x steps (host count, as [8]) of the launches of [9], [13] = of the launches of
 *        [11].  The last launch of an output interval runs bin_every mod 16 model steps when that is not 0, its
 *        predecessor 16: compare the two per particle-step, [9] - [11] * [12] / [13] estimates what the epilogues cost
 *        ([9] - [11] does so only when bin_every is a multiple of the fused step count); accumulated since lpm_set_timing. */
int32_t lpm_get_timing(lpm_handle *h, double *out_host /* [14] */);
/* Number of concentration cells that hold at least one particle in the current binning (the footprint the binning
 * atomics spread over: bench.py measures its atomic peak over exactly that many cells).  Synchronises.
 * Errors: STATE (nothing binned yet). */
int32_t lpm_touched_cells(lpm_handle *h, uint64_t *n_host);

/* ---- micro-benchmarks: measured denominators of the rooflines ------------------ */

/* Time one micro-benchmark with CUDA events on `cuda_stream` (after two warm-up launches, `reps`
 * timed launches) and return operations per second in *ops_per_s_host.  `scratch_dev` is a caller
 * buffer of scratch_bytes (contents are overwritten); footprint_bytes <= scratch_bytes is the
 * address range the memory probes spread over.  kind:
 *   LPM_PROBE_FFMA      fp32 FMA lane-operations / s (8 independent chains per thread)
 *   LPM_PROBE_IMAD_LOP  Philox round mix, IMAD.WIDE.U32 + LOP3, lane-operations / s
 *   LPM_PROBE_RED_F64   random-address red.global.add.f64 over the footprint, atomics / s
 *   LPM_PROBE_RED_U32   random-address red.global.add.u32 over the footprint, atomics / s
 *   LPM_PROBE_RED_SAME  every thread adds to ONE double (hottest-cell service rate), atomics / s
 *   LPM_PROBE_ATOMS     conflict-free shared-memory atomicAdd (u32), atomics / s
 *   LPM_PROBE_GATHER    16-byte loads, each lane its own 32-byte sector of an L1-resident window of
 *                       footprint_bytes: L1 sectors / s (the met gather of a decorrelated warp)
 *   LPM_PROBE_SMEM_GATHER  16-byte shared-memory loads, each lane its own texel of a window of footprint_bytes (<= 16 KB)
 *                       staged in shared memory: lane-loads / s (the alternative to the L1 gathers: 8 per trilinear sample)
 *   LPM_PROBE_GATHER32  32-byte loads (ld.global.nc.v8.f32), each lane its own sector of an L1-resident window: sectors / s
 *                       (the z-pair texel gather of the step kernel: 4 per trilinear sample)
 * Errors: INVALID_ARG (null, unknown kind, scratch < 1 MiB), NO_DEVICE, CUDA. */
typedef enum {
    LPM_PROBE_FFMA = 0, LPM_PROBE_IMAD_LOP = 1, LPM_PROBE_RED_F64 = 2, LPM_PROBE_RED_U32 = 3,
    LPM_PROBE_RED_SAME = 4, LPM_PROBE_ATOMS = 5, LPM_PROBE_GATHER = 6, LPM_PROBE_SMEM_GATHER = 7, LPM_PROBE_GATHER32 = 8
} lpm_probe_kind;
int32_t lpm_probe(int32_t kind, uint64_t footprint_bytes, void *scratch_dev, uint64_t scratch_bytes, int32_t reps,
                  double *ops_per_s_host, void *cuda_stream);

/* ---- stand-alone kernels for parity tests (device arrays in, device arrays out) ------------ */

/* Philox4x32-10 (R1): out_dev[4*i..] = philox(key = seed, ctr = (step, stream, pid_lo, pid_hi))
 * for pid = pid0 + i. */
int32_t lpm_test_philox(uint64_t seed, uint64_t step, uint32_t stream, uint64_t pid0, uint64_t n,
                        uint32_t *out_dev, void *cuda_stream);
/* The same four words from NVIDIA's cuRAND device Philox4x32-10 (stream 0): curand_init(seed, subsequence = pid,
 * offset = 4 * step) + curand4() - an implementation independent of both this library and the oracle
 * (SURVEY.md 8(c) P1).  Test only. */
int32_t lpm_test_curand_philox(uint64_t seed, uint64_t step, uint64_t pid0, uint64_t n, uint32_t *out_dev, void *cuda_stream);
/* The three N(0,1) of R3 for the same counters: out_dev[3*i..]. */
int32_t lpm_test_normals(uint64_t seed, uint64_t step, uint64_t pid0, uint64_t n, float *out_dev,
                         void *cuda_stream);
/* R2 + R3 on given raw words: out_dev[3*i..] = the three N(0,1) Box-Muller makes of the four 32-bit
 * words r_dev[4*i..] (so a test can sweep all 2^24 uniforms the step can ever see). */
int32_t lpm_test_box_muller(const uint32_t *r_dev, uint64_t n, float *out_dev, void *cuda_stream);
/* Met sampling R4 at n points: xyz_dev float4 (w ignored), out_dev float4 (u, v, w, Kz). */
int32_t lpm_test_sample(const lpm_meteo *meteo, double t, const void *xyz_dev, uint64_t n,
                        void *out_dev, void *cuda_stream);

/* ---- met sampling for callers that must not allocate device memory -------------------------- */

/* The same operation as lpm_test_sample (R4: "interpolating ... in x, y, z and time" - the wind and Kz a
 * particle at xyz would see at time t), with identical arguments and bit-identical results, but without a single
 * cudaMalloc / cudaFree.  lpm_test_sample needs two temporary device buffers per call (the z-fastest snapshot pair,
 * 32 bytes per met cell, and the time-blended field, 16 bytes per met cell) and gets them from cudaMalloc.  Some users
 * of the sampler cannot do that:
 *   - a process whose device memory is entirely in the hands of another allocator (a framework's caching pool that has
 *     reserved the whole GPU, a fixed MIG / MPS memory budget): a raw cudaMalloc there fails or eats into a budget the
 *     host application has planned to the byte;
 *   - an operational loop (dose forecast next to a running dispersion model) in which other streams must keep going:
 *     cudaMalloc and cudaFree synchronise the whole device, so every call would stall the model.
 * For them the two buffers live in ONE array that is part of the library image itself (a file-scope __device__
 * array of LPM_SAMPLE_STATIC_BYTES = 12 MiB + 256 B): every GPU on which the library's kernels are loaded holds
 * those bytes from module load until the process exits, whether this function is ever called or not.
 *
 *  LIMIT      grid.nx * grid.ny * grid.nz <= LPM_SAMPLE_STATIC_MAX_CELLS (262144, e.g. 128 x 128 x 16).  A larger
 *             met grid is refused with LPM_ERR_WORKSPACE_TOO_SMALL before anything is enqueued (the built-in array
 *             is this call's workspace); use lpm_test_sample or a handle for those.
 *  FIRST CALL on each device looks up the device address of the array (cudaGetSymbolAddress, with that device
 *             current; the address is cached per device ordinal).  That look-up is a set-up step, not stream work:
 *             make the first call on a device ahead of any stream capture you may have in mind, and with the device
 *             you will use current.  Later calls on that device issue only kernel launches and one 16-byte memset.
 *  SHARED     every call on a device uses the same array and finds the previous call's data in it.  The function
 *             re-writes whatever it reads (the one texel that must be zero, the pad behind the blended field, is
 *             cleared on every call), so calls may follow each other on ONE stream in any mix of grids and times.
 *             Two calls whose GPU work overlaps - different streams, different host threads, different handles -
 *             race on the array and return garbage: serialise them yourself.
 *  ASYNC      unlike lpm_test_sample this call does not synchronise: the work is enqueued on `cuda_stream` (NULL =
 *             default stream) and out_dev is valid once that stream has reached the end of it.  meteo->fields_dev,
 *             xyz_dev, out_dev stay the caller's (inputs are only read); z_levels_host is copied before return.
 *  Errors: INVALID_ARG (as lpm_test_sample; nz > 64 with z_levels_host), WORKSPACE_TOO_SMALL (the limit above),
 *  NO_DEVICE, CUDA (including a failed address look-up).  n = 0 is a valid no-op. */
#define LPM_SAMPLE_STATIC_MAX_CELLS 262144
#define LPM_SAMPLE_STATIC_BYTES (48ull * LPM_SAMPLE_STATIC_MAX_CELLS + 256ull)
int32_t lpm_sample_static(const lpm_meteo *meteo, double t, const void *xyz_dev, uint64_t n, void *out_dev,
                          void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* LPM_H_ */
