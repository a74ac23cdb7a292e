/* lpm_oracle.c — fp64 CPU ORACLE of the Lagrangian particle step + binning.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call this file.  It shares no code
 * with the CUDA path (paper_0912_3223_b200/csrc) and includes none of its headers.
 *
 * What it is: the algorithm of arxiv/paper_0912_3223 (Molnar et al.) written out step by
 * step, in the paper's order (sample weather linearly in x, y, z and time ->
 * diffusion coefficient -> move by wind -> move by turbulent diffusion -> test dry and wet
 * deposition -> particle may become inactive at the boundary; every n-th step activities are
 * summed on a rectangular grid), all arithmetic in double.  Where the paper is silent the
 * readings R1..R10 of DESIGN.md §3 are used and named at the spot.
 *
 * Pins (tests/test_oracle_*.py, `-m "not gpu"`): Philox KAT vectors, Box-Muller moments,
 * the exact Gaussian puff / folded normal (P4), 2^(-t/T) decay (P5), mass ledger (P6), affine
 * reproduction of the interpolation (P7), well-mixed reflection (P8), brute-force binning (P9),
 * closed-form deposition (P10, P11), compaction (P12), schedule (P13), independent numpy trace
 * (P14), geometric-series dose of a resting decaying cloud (P15), Bernoulli deposition (P16), Eq.(3) (P17), levels (P18),
 * drift slope (P19), ground decay: airborne + ground = emitted 2^(-t/T) and the sum of separately decayed increments (P20).
 * PARITY UNPINNED (no printed value or implementation exists to compare against): the
 * dry-deposition rate law p_dry = 1-exp(-vd dt/h_dep) and h_dep, and the treatment of ground,
 * top and lateral boundaries (the paper gives none: L84-86 "out of scope of this paper").
 *
 * Build: gcc -O2 -fopenmp -ffp-contract=off -fPIC -shared lpm_oracle.c -o liblpm_oracle.so -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_MAXK 2
#define ORC_NLEDGER 7 /* emitted, airborne, dry, wet, decayed, exited, dep_offgrid */

typedef struct {
    int32_t nx, ny, nz, pad_;
    double x0, y0, z0, dx, dy, dz;
} orc_grid;

typedef struct {
    orc_grid cgrid;      /* concentration grid; the 2-D deposition map is its (x, y) footprint */
    orc_grid mgrid;      /* meteorology grid, values at cell centres                          */
    int32_t nt, K;
    double t0, dt_snap;
    const float *fields; /* borrowed, [nt][nz][ny][nx][4] = (u, v, w, Kz), x fastest          */
    double Kh, H_mix, kz_min;
    double half_life[ORC_MAXK], vd[ORC_MAXK], lambda_wet[ORC_MAXK];
    double dt;
    uint64_t seed;
    uint64_t capacity;
    int32_t boundary_mode; /* 0 OPEN, 1 ABSORB (R7)                                           */
    int32_t compact;       /* 1: stable compaction of exited particles after every step       */
    double h_dep;
    int32_t bin_every, rain_on;
    double rx0, rx1, ry0, ry1, rt0, rt1; /* rain box (R8/G6)                                  */
    double frag_delta;     /* metres: distance to a discontinuity that flags a particle fragile */
    double face_delta;     /* metres: distance to a deposition-map cell face counted as slack   */
    int32_t dep_mode;      /* 0: expected-mass deposition (R8); 1: paper-literal Bernoulli deposition (R11) */
    int32_t kz_mode;       /* 0: Kz is the interpolated gridded field (R4); 1: Eq.(3) per particle (R12)    */
    const float *surface;  /* kz_mode 1: borrowed, [nt][ny][nx][4] = (u*, 1/L, Hz, unused), x fastest         */
    const double *z_levels; /* NULL: uniform levels z0 + (k + 1/2) dz; else borrowed, mgrid.nz ascending heights of
                             * the met levels ("vertical weather information is nonlinear")     */
    int32_t drift;          /* 1: LABELLED DEPARTURE from the paper: z' gets the drift correction
                             * + dKz/dz * dt of the well-mixed random walk; kz_mode 0 only                      */
    int32_t pad3_;
} orc_config;

typedef struct {
    double x, y, z, t_start, t_end;
    double total_activity[ORC_MAXK];
    uint64_t n_particles; /* count mode if > 0 */
    double rate;          /* particles per second otherwise */
    uint64_t pid_offset, pid_stride;
} orc_source;

typedef struct {
    orc_source src;
    int64_t s_start, S; /* first release step, number of release steps */
    uint64_t c;         /* rate mode: slots per step                   */
    uint64_t next_l;    /* count mode: next local index to be born     */
} orc_rel;

typedef struct orc_sim {
    orc_config cfg;
    float p_dry[ORC_MAXK], p_wet[ORC_MAXK]; /* fp32 parameters (R8) */
    double f_decay[ORC_MAXK];
    float sigma_h;                          /* fp32 parameter (R5)  */
    uint64_t step;
    /* particles */
    uint64_t n, cap;
    double *x, *y, *z, *m[ORC_MAXK];
    uint64_t *pid;
    uint8_t *status;  /* 0 active, 1 exited */
    uint8_t *fragile;
    /* per-step scratch */
    double *inc_dry[ORC_MAXK], *inc_wet[ORC_MAXK], *inc_dec[ORC_MAXK];
    int64_t *dcell;   /* deposition cell of the new position, -1 = off the map */
    uint8_t *nearface; /* bit0: near lower-x face, bit1 upper-x, bit2 lower-y, bit3 upper-y */
    uint8_t *moved;
    /* releases */
    orc_rel rel[8];
    int32_t n_rel;
    /* outputs */
    double ledger[ORC_MAXK][ORC_NLEDGER];
    double *conc_sum; /* [K][nz][ny][nx] sum of activity per cell at the last binning */
    uint32_t *cnt;    /* [nz][ny][nx] */
    double *dep;      /* [K][ny][nx] cumulative deposited activity */
    double *dep_slack;
    uint64_t *inj_log; uint64_t inj_cap;
    uint64_t *frag_pids; uint64_t n_frag, frag_cap; /* pids ever flagged fragile (T3) */
    uint64_t bin_step;
    double *dose;     /* [K][nz][ny][nx] time-integrated concentration, Bq s m^-3; NULL = not accumulated */
    double *ground, *ground_slack; /* [K][ny][nx] deposited activity that keeps decaying on the ground (R13); NULL = off */
} orc_sim;

/* ------------------------------------------------------------------ R1: Philox4x32-10
 * Salmon, Moraes, Dror, Shaw, "Parallel random numbers: as easy as 1, 2, 3" (SC'11): the
 * counter-based generator named by BASELINE.json north_star in place of the paper's Mersenne
 * Twister.  Round: (c0,c1,c2,c3) <- (hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1,
 * lo(M0*c0)); the key is bumped by the Weyl constants between rounds; 10 rounds. */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
    for (int r = 0; r < 10; ++r) {
        uint64_t p0 = (uint64_t)M0 * c0, p1 = (uint64_t)M1 * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += W0; k1 += W1;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* counter layout (R1): key = (seed_lo, seed_hi), ctr = (step, stream, pid_lo, pid_hi) */
void orc_philox_draw(uint64_t seed, uint64_t pid, uint64_t step, uint32_t stream, uint32_t out[4])
{
    uint32_t ctr[4] = {(uint32_t)step, stream, (uint32_t)pid, (uint32_t)(pid >> 32)};
    uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
    orc_philox4x32_10(ctr, key, out);
}

/* R2: four exact 24-bit uniforms; u[0], u[2] in (0,1] (log arguments), u[1], u[3] in [0,1) */
void orc_uniforms(const uint32_t r[4], double u[4])
{
    const double s = 1.0 / 16777216.0;
    u[0] = ((double)(r[0] >> 8) + 1.0) * s;
    u[1] = (double)(r[1] >> 8) * s;
    u[2] = ((double)(r[2] >> 8) + 1.0) * s;
    u[3] = (double)(r[3] >> 8) * s;
}

/* R3: basic (trigonometric) Box-Muller, PAPER.md L77 ref [37]; fixed 4-in / 3-out budget */
void orc_normals(uint64_t seed, uint64_t pid, uint64_t step, double nrm[3])
{
    uint32_t r[4];
    double u[4];
    const double two_pi = 6.283185307179586476925286766559;
    orc_philox_draw(seed, pid, step, 0u, r);
    orc_uniforms(r, u);
    double R1 = sqrt(-2.0 * log(u[0])), R2 = sqrt(-2.0 * log(u[2]));
    nrm[0] = R1 * cos(two_pi * u[1]);
    nrm[1] = R1 * sin(two_pi * u[1]);
    nrm[2] = R2 * cos(two_pi * u[3]);
}

/* ------------------------------------------------------------------ R4: met sampling
 * "interpolating (sampling) weather data in x, y, z, and time dimensions using
 * linear interpolation".  Cell-centred values, edge-clamped (paper silent on the edges). */
static void axis_weights(double p, double p0, double dp, int32_t n, int32_t *i0, int32_t *i1, double *f)
{
    double g = (p - p0) / dp - 0.5;
    if (g < 0.0) g = 0.0;
    if (g > (double)(n - 1)) g = (double)(n - 1);
    int32_t lo = (int32_t)floor(g);
    int32_t lim = n - 2 > 0 ? n - 2 : 0;
    if (lo > lim) lo = lim;
    *i0 = lo;
    *i1 = lo + 1 < n - 1 ? lo + 1 : n - 1;
    *f = g - (double)lo;
}

/* non-uniform levels (L110): linear between the two levels that bracket z, clamped below the first and above
 * the last level; k0 = the last level at or below z, at most n - 2 */
static void level_weights(double z, const double *zl, int32_t n, int32_t *k0, int32_t *k1, double *f)
{
    if (n < 2) { *k0 = *k1 = 0; *f = 0.0; return; }
    int32_t k = 0;
    while (k < n - 2 && zl[k + 1] <= z) ++k;
    double w = (z - zl[k]) / (zl[k + 1] - zl[k]);
    if (w < 0.0) w = 0.0;
    if (w > 1.0) w = 1.0;
    *k0 = k; *k1 = k + 1; *f = w;
}

static void sample_snapshot(const orc_grid *g, const double *levels, const float *snap, double x, double y, double z, double out[4])
{
    int32_t i0, i1, j0, j1, k0, k1;
    double fx, fy, fz;
    axis_weights(x, g->x0, g->dx, g->nx, &i0, &i1, &fx);
    axis_weights(y, g->y0, g->dy, g->ny, &j0, &j1, &fy);
    if (levels) level_weights(z, levels, g->nz, &k0, &k1, &fz);
    else axis_weights(z, g->z0, g->dz, g->nz, &k0, &k1, &fz);
    const int32_t I[2] = {i0, i1}, J[2] = {j0, j1}, Kk[2] = {k0, k1};
    const double wx[2] = {1.0 - fx, fx}, wy[2] = {1.0 - fy, fy}, wz[2] = {1.0 - fz, fz};
    for (int c = 0; c < 4; ++c) out[c] = 0.0;
    for (int kk = 0; kk < 2; ++kk)
        for (int jj = 0; jj < 2; ++jj)
            for (int ii = 0; ii < 2; ++ii) {
                size_t cell = ((size_t)Kk[kk] * g->ny + J[jj]) * g->nx + I[ii];
                double w = wz[kk] * wy[jj] * wx[ii];
                for (int c = 0; c < 4; ++c) out[c] += w * (double)snap[4 * cell + c];
            }
}

/* SURVEY 8(f)4, not in the paper: d/dz of the trilinear interpolant of component 3 (Kz) of one snapshot at (x, y, z):
 * the slope between the two bracketing levels, weighted bilinearly in x and y; 0 outside the open hull of the
 * level heights (where the interpolant is clamped, i.e. constant in z) and on a single-level grid. */
static double snapshot_dkz_dz(const orc_grid *g, const double *levels, const float *snap, double x, double y, double z)
{
    int32_t i0, i1, j0, j1, k0, k1;
    double fx, fy, fz, lo, hi, h;
    if (g->nz < 2) return 0.0;
    if (levels) { lo = levels[0]; hi = levels[g->nz - 1]; }
    else { lo = g->z0 + 0.5 * g->dz; hi = g->z0 + ((double)g->nz - 0.5) * g->dz; }
    if (!(z > lo && z < hi)) return 0.0;
    axis_weights(x, g->x0, g->dx, g->nx, &i0, &i1, &fx);
    axis_weights(y, g->y0, g->dy, g->ny, &j0, &j1, &fy);
    if (levels) { level_weights(z, levels, g->nz, &k0, &k1, &fz); h = levels[k1] - levels[k0]; }
    else { axis_weights(z, g->z0, g->dz, g->nz, &k0, &k1, &fz); h = g->dz; }
    const int32_t I[2] = {i0, i1}, J[2] = {j0, j1};
    const double wx[2] = {1.0 - fx, fx}, wy[2] = {1.0 - fy, fy};
    double d = 0.0;
    for (int jj = 0; jj < 2; ++jj)
        for (int ii = 0; ii < 2; ++ii) {
            size_t c0 = ((size_t)k0 * g->ny + J[jj]) * g->nx + I[ii], c1 = ((size_t)k1 * g->ny + J[jj]) * g->nx + I[ii];
            d += wy[jj] * wx[ii] * ((double)snap[4 * c1 + 3] - (double)snap[4 * c0 + 3]);
        }
    return d / h;
}

/* time weight: s = clamp(floor((t-t0)/dT), 0, nt-2); a = clamp((t-T_s)/dT, 0, 1), rounded to
 * fp32 (the fp32 value is the parameter of both sides, DESIGN.md §3 R4). nt == 1: s = 0, a = 0. */
void orc_time_weight(int32_t nt, double t0, double dt_snap, double t, int32_t *s_out, float *a_out)
{
    if (nt <= 1) { *s_out = 0; *a_out = 0.0f; return; }
    double r = floor((t - t0) / dt_snap);
    if (r < 0.0) r = 0.0;
    if (r > (double)(nt - 2)) r = (double)(nt - 2);
    int32_t s = (int32_t)r;
    double a = (t - (t0 + (double)s * dt_snap)) / dt_snap;
    if (a < 0.0) a = 0.0;
    if (a > 1.0) a = 1.0;
    *s_out = s;
    *a_out = (float)a;
}

/* levels == NULL: uniform vertical levels (R4); else the nz ascending level heights (L110) */
void orc_sample_met_levels(const orc_grid *g, const double *levels, int32_t nt, double t0, double dt_snap, const float *fields,
                           double t, double x, double y, double z, double out[4])
{
    int32_t s; float a;
    size_t snap_elems = (size_t)g->nx * g->ny * g->nz * 4;
    orc_time_weight(nt, t0, dt_snap, t, &s, &a);
    double A[4], B[4];
    sample_snapshot(g, levels, fields + (size_t)s * snap_elems, x, y, z, A);
    if (nt > 1) {
        sample_snapshot(g, levels, fields + (size_t)(s + 1) * snap_elems, x, y, z, B);
        for (int c = 0; c < 4; ++c) out[c] = (1.0 - (double)a) * A[c] + (double)a * B[c];
    } else {
        for (int c = 0; c < 4; ++c) out[c] = A[c];
    }
}

double orc_dkz_dz(const orc_grid *g, const double *levels, int32_t nt, double t0, double dt_snap, const float *fields, double t,
                  double x, double y, double z)
{
    int32_t s; float a;
    size_t snap_elems = (size_t)g->nx * g->ny * g->nz * 4;
    orc_time_weight(nt, t0, dt_snap, t, &s, &a);
    double d0 = snapshot_dkz_dz(g, levels, fields + (size_t)s * snap_elems, x, y, z);
    if (nt <= 1) return d0;
    double d1 = snapshot_dkz_dz(g, levels, fields + (size_t)(s + 1) * snap_elems, x, y, z);
    return (1.0 - (double)a) * d0 + (double)a * d1;
}

void orc_sample_met(const orc_grid *g, int32_t nt, double t0, double dt_snap, const float *fields,
                    double t, double x, double y, double z, double out[4])
{
    orc_sample_met_levels(g, NULL, nt, t0, dt_snap, fields, t, x, y, z, out);
}

/* ------------------------------------------------------------------ R12: Eq.(3) per particle
 * PAPER.md L79-82 Eq.(3): Kz(z) = k u* z / Phi(z/L) * (1 - z/Hz)^2, "where k, u*, z, Phi, L and Hz are the von
 * Karman constant, friction velocity, height, stability function, Monin-Obukhov length and mixing layer
 * height".  The paper defines no Phi (G2); reading R12 takes the Businger-Dyer forms
 * Phi = 1 + 5 zeta (zeta = z/L >= 0), Phi = (1 - 16 zeta)^(-1/2) (zeta < 0), k = 0.4, Kz = 0 at and above Hz.
 * u*, 1/L and Hz are 2-D fields sampled like the weather (L106: linear in x, y and time; cell-centred,
 * edge-clamped as R4); 1/L, not L, is the stored and interpolated quantity (neutral = 0). */
void orc_sample_surface(const orc_grid *g, int32_t nt, double t0, double dt_snap, const float *surface, double t, double x,
                        double y, double out[3])
{
    int32_t s, i0, i1, j0, j1;
    float a;
    double fx, fy;
    orc_time_weight(nt, t0, dt_snap, t, &s, &a);
    axis_weights(x, g->x0, g->dx, g->nx, &i0, &i1, &fx);
    axis_weights(y, g->y0, g->dy, g->ny, &j0, &j1, &fy);
    const size_t plane = (size_t)g->nx * g->ny * 4;
    for (int c = 0; c < 3; ++c) {
        double v[2] = {0.0, 0.0};
        for (int tt = 0; tt < (nt > 1 ? 2 : 1); ++tt) {
            const float *f = surface + (size_t)(s + tt) * plane;
            v[tt] = (1.0 - fy) * ((1.0 - fx) * (double)f[4 * ((size_t)j0 * g->nx + i0) + c] + fx * (double)f[4 * ((size_t)j0 * g->nx + i1) + c]) +
                    fy * ((1.0 - fx) * (double)f[4 * ((size_t)j1 * g->nx + i0) + c] + fx * (double)f[4 * ((size_t)j1 * g->nx + i1) + c]);
        }
        out[c] = nt > 1 ? (1.0 - (double)a) * v[0] + (double)a * v[1] : v[0];
    }
}

double orc_kz_eq3(double ustar, double inv_L, double Hz, double z)
{
    if (!(z < Hz) || !(z > 0.0)) return 0.0;
    double zeta = z * inv_L;
    double phi = zeta >= 0.0 ? 1.0 + 5.0 * zeta : 1.0 / sqrt(1.0 - 16.0 * zeta);
    double t = 1.0 - z / Hz;
    return 0.4 * ustar * z / phi * t * t;
}

/* ------------------------------------------------------------------ R10: cell index
 * Defined in fp32, exactly: i = (int)floorf((x - x0) * inv_dx), inv_dx = (float)(1.0/dx).
 * The expression has no a*b+c shape, so FMA contraction cannot alter it (and this file is
 * compiled with -ffp-contract=off).  Returns -1 when outside [0, n). */
int32_t orc_cell_index(float p, double p0, double dp, int32_t n)
{
    volatile float o = (float)p0;
    volatile float inv = (float)(1.0 / dp);
    volatile float d = p - o;
    volatile float s = d * inv;
    float fl = floorf(s);
    if (!(fl >= 0.0f) || !(fl < (float)n)) return -1;
    return (int32_t)fl;
}

/* ------------------------------------------------------------------ simulation object */
static void *xrealloc(void *p, size_t bytes) { void *q = realloc(p, bytes ? bytes : 1); if (!q) abort(); return q; }

static void grow(orc_sim *s, uint64_t need)
{
    if (need <= s->cap) return;
    uint64_t nc = s->cap ? s->cap : 1024;
    while (nc < need) nc *= 2;
    s->x = xrealloc(s->x, nc * sizeof(double));
    s->y = xrealloc(s->y, nc * sizeof(double));
    s->z = xrealloc(s->z, nc * sizeof(double));
    s->pid = xrealloc(s->pid, nc * sizeof(uint64_t));
    s->status = xrealloc(s->status, nc);
    s->fragile = xrealloc(s->fragile, nc);
    s->dcell = xrealloc(s->dcell, nc * sizeof(int64_t));
    s->nearface = xrealloc(s->nearface, nc);
    s->moved = xrealloc(s->moved, nc);
    for (int k = 0; k < ORC_MAXK; ++k) {
        s->m[k] = xrealloc(s->m[k], nc * sizeof(double));
        s->inc_dry[k] = xrealloc(s->inc_dry[k], nc * sizeof(double));
        s->inc_wet[k] = xrealloc(s->inc_wet[k], nc * sizeof(double));
        s->inc_dec[k] = xrealloc(s->inc_dec[k], nc * sizeof(double));
    }
    s->cap = nc;
}

orc_sim *orc_create(const orc_config *cfg)
{
    if (!cfg || cfg->K < 1 || cfg->K > ORC_MAXK || cfg->nt < 1 || !(cfg->dt > 0.0)) return NULL;
    orc_sim *s = calloc(1, sizeof(orc_sim));
    if (!s) return NULL;
    s->cfg = *cfg;
    /* R5: sigma_h = sqrt(2 Kh dt) (Eq.(2)), an fp32 parameter of both sides */
    s->sigma_h = (float)sqrt(2.0 * cfg->Kh * cfg->dt);
    for (int k = 0; k < cfg->K; ++k) {
        /* R8: per-step removal probabilities, computed in double, rounded once to fp32 */
        s->p_dry[k] = (cfg->vd[k] > 0.0 && cfg->h_dep > 0.0) ? (float)(-expm1(-cfg->vd[k] * cfg->dt / cfg->h_dep)) : 0.0f;
        s->p_wet[k] = (cfg->lambda_wet[k] > 0.0) ? (float)(-expm1(-cfg->lambda_wet[k] * cfg->dt)) : 0.0f;
        /* decay "deterministic ... based on half-time": exp(-ln2 dt / T_half) */
        s->f_decay[k] = cfg->half_life[k] > 0.0 ? exp(-M_LN2 * cfg->dt / cfg->half_life[k]) : 1.0;
    }
    const orc_grid *g = &s->cfg.cgrid;
    size_t cells3 = (size_t)g->nx * g->ny * g->nz, cells2 = (size_t)g->nx * g->ny;
    s->conc_sum = calloc(cells3 * cfg->K, sizeof(double));
    s->cnt = calloc(cells3, sizeof(uint32_t));
    s->dep = calloc(cells2 * cfg->K, sizeof(double));
    s->dep_slack = calloc(cells2 * cfg->K, sizeof(double));
    if (!s->conc_sum || !s->cnt || !s->dep || !s->dep_slack) abort();
    return s;
}

void orc_destroy(orc_sim *s)
{
    if (!s) return;
    free(s->x); free(s->y); free(s->z); free(s->pid); free(s->status); free(s->fragile);
    free(s->dcell); free(s->nearface); free(s->moved);
    for (int k = 0; k < ORC_MAXK; ++k) { free(s->m[k]); free(s->inc_dry[k]); free(s->inc_wet[k]); free(s->inc_dec[k]); }
    free(s->conc_sum); free(s->cnt); free(s->dep); free(s->dep_slack); free(s->inj_log); free(s->frag_pids); free(s->dose); free(s->ground); free(s->ground_slack);
    free(s);
}

/* R9: release schedule ("released ... in each time step", L104 a-priori assignment
 * of activity, L128 "emission is always scaled to the given total number of particles"). */
int32_t orc_release(orc_sim *s, const orc_source *src)
{
    if (!s || !src || s->n_rel >= 8) return -1;
    if (src->pid_stride < 1) return -1;
    orc_rel *r = &s->rel[s->n_rel];
    memset(r, 0, sizeof(*r));
    r->src = *src;
    r->s_start = (int64_t)ceil(src->t_start / s->cfg.dt);
    r->S = (int64_t)ceil((src->t_end - src->t_start) / s->cfg.dt);
    if (r->S < 1) r->S = 1;
    if (src->n_particles == 0) {
        if (src->pid_stride != 1) return -1;
        r->c = (uint64_t)llround(src->rate * s->cfg.dt);
        if (r->c == 0) return -1;
    }
    if ((int64_t)s->step > r->s_start) return -1; /* releases must be registered before they start */
    s->n_rel++;
    return 0;
}

static void birth(orc_sim *s, const orc_rel *r, uint64_t pid, double denom)
{
    grow(s, s->n + 1);
    uint64_t i = s->n++;
    s->x[i] = r->src.x; s->y[i] = r->src.y; s->z[i] = r->src.z;
    s->pid[i] = pid; s->status[i] = 0; s->fragile[i] = 0;
    for (int k = 0; k < s->cfg.K; ++k) {
        double m = r->src.total_activity[k] / denom; /* activity a priori assigned, L104 */
        s->m[k][i] = m;
        s->ledger[k][0] += m;
    }
}

static void inject(orc_sim *s, uint64_t n)
{
    uint64_t injected = 0;
    for (int ri = 0; ri < s->n_rel; ++ri) {
        orc_rel *r = &s->rel[ri];
        int64_t rs = (int64_t)n - r->s_start;
        if (rs < 0) continue;
        if (r->src.n_particles > 0) {
            /* count mode: global particle j of N is born at step s_start + floor(j*S/N) */
            uint64_t N = r->src.n_particles;
            for (;;) {
                uint64_t j = r->src.pid_offset + r->next_l * r->src.pid_stride;
                if (j >= N) break;
                int64_t b = r->s_start + (int64_t)(((unsigned __int128)j * (uint64_t)r->S) / N);
                if (b > (int64_t)n) break;
                birth(s, r, j, (double)N);
                r->next_l++; injected++;
            }
        } else if (rs < r->S) {
            /* rate mode: c slots per step, pid = offset + (n - s_start)*c + j; when capacity is
             * short the highest j are skipped and never renumbered */
            uint64_t room = s->cfg.capacity > s->n ? s->cfg.capacity - s->n : 0;
            uint64_t take = r->c < room ? r->c : room;
            for (uint64_t j = 0; j < take; ++j)
                birth(s, r, r->src.pid_offset + (uint64_t)rs * r->c + j, (double)r->c * (double)r->S);
            injected += take;
        }
    }
    if (n >= s->inj_cap) {
        uint64_t nc = s->inj_cap ? s->inj_cap * 2 : 1024;
        while (nc <= n) nc *= 2;
        s->inj_log = xrealloc(s->inj_log, nc * sizeof(uint64_t));
        memset(s->inj_log + s->inj_cap, 0, (nc - s->inj_cap) * sizeof(uint64_t));
        s->inj_cap = nc;
    }
    s->inj_log[n] = injected;
}

/* ------------------------------------------------------------------ one particle, one step
 * Order of operations: PAPER.md L106-108.  Eq.(1): X_new = X_old + v_adv dt + x~ (L71);
 * Eq.(2): x~_i = rand * sqrt(2 K_i dt) (L75). */
static void step_particle(orc_sim *s, uint64_t i, uint64_t n, double t_n, int raining)
{
    const orc_config *c = &s->cfg;
    double nrm[3], met[4];
    s->moved[i] = 0;
    s->dcell[i] = -1;
    s->nearface[i] = 0;
    for (int k = 0; k < c->K; ++k) s->inc_dry[k][i] = s->inc_wet[k][i] = s->inc_dec[k][i] = 0.0;
    if (s->status[i] != 0) return;
    s->moved[i] = 1;

    /* R1-R3: three N(0,1) draws from Philox stream 0 keyed by (seed, pid, step) */
    orc_normals(c->seed, s->pid[i], n, nrm);

    /* R4: weather at X_old, t_n (forward Euler; Eq.(1) uses the wind at the old position) */
    orc_sample_met_levels(&c->mgrid, c->z_levels, c->nt, c->t0, c->dt_snap, c->fields, t_n, s->x[i], s->y[i], s->z[i], met);
    double u = met[0], v = met[1], w = met[2], Kz = met[3];
    if (c->kz_mode == 1) { /* R12: "computing the turbulent diffusion coefficient" per particle (L106, L112-113) */
        double sf[3];
        orc_sample_surface(&c->mgrid, c->nt, c->t0, c->dt_snap, c->surface, t_n, s->x[i], s->y[i], sf);
        Kz = orc_kz_eq3(sf[0], sf[1], sf[2], s->z[i]);
    }
    double drift = 0.0;
    if (c->drift == 1 && c->kz_mode == 0 && !(Kz < c->kz_min)) { /* SURVEY 8(f)4 departure; a floored Kz is constant in z */
        drift = orc_dkz_dz(&c->mgrid, c->z_levels, c->nt, c->t0, c->dt_snap, c->fields, t_n, s->x[i], s->y[i], s->z[i]) * c->dt;
        const orc_grid *mg = &c->mgrid;
        double zlo = c->z_levels ? c->z_levels[0] : mg->z0 + 0.5 * mg->dz;
        double zhi = c->z_levels ? c->z_levels[mg->nz - 1] : mg->z0 + ((double)mg->nz - 0.5) * mg->dz;
        if (fabs(s->z[i] - zlo) < c->frag_delta || fabs(s->z[i] - zhi) < c->frag_delta) { if (s->fragile[i] == 0) s->fragile[i] = 1; } /* slope switches on / off there */
    }
    if (Kz < c->kz_min) Kz = c->kz_min;

    /* R5: Eq.(1) + Eq.(2) */
    double xn = s->x[i] + u * c->dt + (double)s->sigma_h * nrm[0];
    double yn = s->y[i] + v * c->dt + (double)s->sigma_h * nrm[1];
    double zn = s->z[i] + w * c->dt + drift + sqrt(2.0 * Kz * c->dt) * nrm[2];

    /* R6: reflection at the ground and at the mixing height (north_star; paper silent) */
    if (zn < 0.0) zn = -zn;
    if (zn > c->H_mix) zn = 2.0 * c->H_mix - zn;
    if (zn < 0.0) zn = 0.0;

    s->x[i] = xn; s->y[i] = yn; s->z[i] = zn;

    /* R7: lateral boundary = met-grid box ("reaches the predefined boundaries") */
    const orc_grid *g = &c->mgrid;
    double bx0 = g->x0, bx1 = g->x0 + g->nx * g->dx, by0 = g->y0, by1 = g->y0 + g->ny * g->dy;
    if (c->boundary_mode == 1) {
        double dmin = fmin(fmin(fabs(xn - bx0), fabs(xn - bx1)), fmin(fabs(yn - by0), fabs(yn - by1)));
        if (dmin < c->frag_delta) { if (s->fragile[i] == 0) s->fragile[i] = 1; }
        if (!(xn >= bx0 && xn < bx1 && yn >= by0 && yn < by1)) {
            s->status[i] = 1;
            return; /* mass is moved to the exited ledger by the serial pass */
        }
    }

    /* R8: deposition, then decay, at the new position */
    int eligible = (c->h_dep >= c->H_mix) || (zn < c->h_dep);
    if (c->h_dep < c->H_mix && fabs(zn - c->h_dep) < c->frag_delta) { if (s->fragile[i] == 0) s->fragile[i] = 1; }
    int wet = 0;
    if (raining) {
        wet = (xn >= c->rx0 && xn < c->rx1 && yn >= c->ry0 && yn < c->ry1);
        /* distance to the rectangle's boundary */
        double ddx = fmin(fabs(xn - c->rx0), fabs(xn - c->rx1));
        double ddy = fmin(fabs(yn - c->ry0), fabs(yn - c->ry1));
        int near_x = ddx < c->frag_delta && yn >= c->ry0 - c->frag_delta && yn <= c->ry1 + c->frag_delta;
        int near_y = ddy < c->frag_delta && xn >= c->rx0 - c->frag_delta && xn <= c->rx1 + c->frag_delta;
        if (near_x || near_y) { if (s->fragile[i] == 0) s->fragile[i] = 1; }
    }
    int any = 0;
    if (c->dep_mode == 1) {
        /* R11, the paper's own form ("deposition ... considered stochastic", L114 "testing for
         * dry and wet depositions", L108 a deposited particle becomes inactive): one Bernoulli trial per
         * nuclide and sink per step, from Philox stream 1 of the same (seed, id, step): word k decides dry,
         * word 2 + k decides wet deposition of nuclide k; u = (word >> 8) 2^-24 in [0, 1), event iff u < p
         * (p the fp32 parameter of R8; the comparison is exact on both sides).  The event deposits the
         * nuclide's WHOLE activity at the new (x, y); dry is tried first, wet only if dry did not fire. */
        uint32_t r1[4];
        orc_philox_draw(c->seed, s->pid[i], n, 1u, r1);
        const double sc = 1.0 / 16777216.0;
        for (int k = 0; k < c->K; ++k) {
            double m = s->m[k][i], dd = 0.0, dw = 0.0;
            if (m > 0.0) {
                double ud = (double)(r1[k] >> 8) * sc, uw = (double)(r1[2 + k] >> 8) * sc;
                if (eligible && ud < (double)s->p_dry[k]) { dd = m; m = 0.0; }
                else if (wet && uw < (double)s->p_wet[k]) { dw = m; m = 0.0; }
            }
            double mn = m * s->f_decay[k];
            s->inc_dry[k][i] = dd; s->inc_wet[k][i] = dw; s->inc_dec[k][i] = m - mn;
            s->m[k][i] = mn;
            if (dd != 0.0 || dw != 0.0) any = 1;
        }
        int empty = 1;
        for (int k = 0; k < c->K; ++k) if (s->m[k][i] > 0.0) empty = 0;
        if (empty) s->status[i] = 2; /* deposited: inactive from now on (L108) */
    } else
    for (int k = 0; k < c->K; ++k) {
        double m = s->m[k][i];
        double dd = eligible ? m * (double)s->p_dry[k] : 0.0;
        m -= dd;
        double dw = wet ? m * (double)s->p_wet[k] : 0.0;
        m -= dw;
        double mn = m * s->f_decay[k];
        s->inc_dry[k][i] = dd; s->inc_wet[k][i] = dw; s->inc_dec[k][i] = m - mn;
        s->m[k][i] = mn;
        if (dd != 0.0 || dw != 0.0) any = 1;
    }
    if (any) {
        /* deposition cell of the NEW (x, y), by the fp32 index rule R10 */
        const orc_grid *cg = &c->cgrid;
        float xf = (float)xn, yf = (float)yn;
        int32_t ci = orc_cell_index(xf, cg->x0, cg->dx, cg->nx);
        int32_t cj = orc_cell_index(yf, cg->y0, cg->dy, cg->ny);
        if (ci >= 0 && cj >= 0) s->dcell[i] = (int64_t)cj * cg->nx + ci;
        else s->dcell[i] = -2; /* deposited off the map */
        double gxp = (xn - cg->x0) / cg->dx, gyp = (yn - cg->y0) / cg->dy;
        double fxp = gxp - floor(gxp), fyp = gyp - floor(gyp);
        uint8_t nf = 0;
        if (fxp * cg->dx < c->face_delta) nf |= 1;
        if ((1.0 - fxp) * cg->dx < c->face_delta) nf |= 2;
        if (fyp * cg->dy < c->face_delta) nf |= 4;
        if ((1.0 - fyp) * cg->dy < c->face_delta) nf |= 8;
        s->nearface[i] = nf;
    }
}

static void add_slack(orc_sim *s, int k, int64_t ci, int64_t cj, double v)
{
    const orc_grid *cg = &s->cfg.cgrid;
    if (ci < 0 || cj < 0 || ci >= cg->nx || cj >= cg->ny) return;
    s->dep_slack[((size_t)k * cg->ny + cj) * cg->nx + ci] += v;
    if (s->ground_slack) s->ground_slack[((size_t)k * cg->ny + cj) * cg->nx + ci] += v;
}

/* R10 / PAPER.md L108: "Activities or masses of particles are summarized on a rectangular grid" */
void orc_bin_now(orc_sim *s)
{
    const orc_grid *g = &s->cfg.cgrid;
    size_t cells3 = (size_t)g->nx * g->ny * g->nz;
    memset(s->conc_sum, 0, cells3 * s->cfg.K * sizeof(double));
    memset(s->cnt, 0, cells3 * sizeof(uint32_t));
    for (uint64_t i = 0; i < s->n; ++i) {
        if (s->status[i] != 0) continue;
        int32_t ci = orc_cell_index((float)s->x[i], g->x0, g->dx, g->nx);
        int32_t cj = orc_cell_index((float)s->y[i], g->y0, g->dy, g->ny);
        int32_t ck = orc_cell_index((float)s->z[i], g->z0, g->dz, g->nz);
        if (ci < 0 || cj < 0 || ck < 0) continue;
        size_t cell = ((size_t)ck * g->ny + cj) * g->nx + ci;
        s->cnt[cell] += 1u;
        for (int k = 0; k < s->cfg.K; ++k) s->conc_sum[(size_t)k * cells3 + cell] += s->m[k][i];
    }
    s->bin_step = s->step;
}

int32_t orc_step(orc_sim *s, int32_t n_steps)
{
    if (!s || n_steps < 0) return -1;
    const orc_config *c = &s->cfg;
    const orc_grid *cg = &c->cgrid;
    for (int32_t it = 0; it < n_steps; ++it) {
        uint64_t n = s->step;
        double t_n = (double)n * c->dt;
        inject(s, n);
        int raining = c->rain_on && t_n >= c->rt0 && t_n < c->rt1; /* G6: tested at t_n */
        int64_t cnt = (int64_t)s->n;
#pragma omp parallel for schedule(static)
        for (int64_t i = 0; i < cnt; ++i) step_particle(s, (uint64_t)i, n, t_n, raining);

        /* serial fp64 accumulation of the deposit map and the ledger, in particle order */
        for (uint64_t i = 0; i < s->n; ++i) {
            if (!s->moved[i]) continue;
            if (s->fragile[i] == 1) {
                if (s->n_frag == s->frag_cap) {
                    s->frag_cap = s->frag_cap ? 2 * s->frag_cap : 256;
                    s->frag_pids = xrealloc(s->frag_pids, s->frag_cap * sizeof(uint64_t));
                }
                s->frag_pids[s->n_frag++] = s->pid[i];
                s->fragile[i] = 2;
            }
            if (s->status[i] == 1) {
                for (int k = 0; k < c->K; ++k) { s->ledger[k][5] += s->m[k][i]; s->m[k][i] = 0.0; }
                continue;
            }
            /* status 2 (deposited in this step, R11) falls through: its increments are booked below */
            for (int k = 0; k < c->K; ++k) {
                double d = s->inc_dry[k][i] + s->inc_wet[k][i];
                s->ledger[k][2] += s->inc_dry[k][i];
                s->ledger[k][3] += s->inc_wet[k][i];
                s->ledger[k][4] += s->inc_dec[k][i];
                if (d == 0.0) continue;
                if (s->dcell[i] >= 0) {
                    s->dep[(size_t)k * cg->nx * cg->ny + (size_t)s->dcell[i]] += d;
                    if (s->ground) s->ground[(size_t)k * cg->nx * cg->ny + (size_t)s->dcell[i]] += d;
                    int64_t ci = s->dcell[i] % cg->nx, cj = s->dcell[i] / cg->nx;
                    uint8_t nf = s->nearface[i];
                    if (nf) {
                        add_slack(s, k, ci, cj, d);
                        if (nf & 1) add_slack(s, k, ci - 1, cj, d);
                        if (nf & 2) add_slack(s, k, ci + 1, cj, d);
                        if (nf & 4) add_slack(s, k, ci, cj - 1, d);
                        if (nf & 8) add_slack(s, k, ci, cj + 1, d);
                        if ((nf & 1) && (nf & 4)) add_slack(s, k, ci - 1, cj - 1, d);
                        if ((nf & 1) && (nf & 8)) add_slack(s, k, ci - 1, cj + 1, d);
                        if ((nf & 2) && (nf & 4)) add_slack(s, k, ci + 1, cj - 1, d);
                        if ((nf & 2) && (nf & 8)) add_slack(s, k, ci + 1, cj + 1, d);
                    }
                } else {
                    s->ledger[k][6] += d;
                    /* a particle just outside the map may have been inside on the other side */
                    if (s->nearface[i]) {
                        double gxp = floor((s->x[i] - cg->x0) / cg->dx), gyp = floor((s->y[i] - cg->y0) / cg->dy);
                        for (int dj = -1; dj <= 1; ++dj) for (int di = -1; di <= 1; ++di)
                            add_slack(s, k, (int64_t)gxp + di, (int64_t)gyp + dj, d);
                    }
                }
            }
        }
        /* R13 (SURVEY 8(c) R8 "a read-out-time option", 8(f)3 "ground-decay of the deposition map"): what lies on the
         * ground decays like what is in the air.  The increments of step n were evaluated at t_n (R8: the mass at the
         * start of the step), so they decay over this step too: ground(t_{n+1}) = (ground(t_n) + increments) exp(-lambda dt) */
        if (s->ground) {
            size_t c2 = (size_t)cg->nx * cg->ny;
            for (int k = 0; k < c->K; ++k)
                for (size_t i = 0; i < c2; ++i) {
                    s->ground[(size_t)k * c2 + i] *= s->f_decay[k];
                    s->ground_slack[(size_t)k * c2 + i] *= s->f_decay[k];
                }
        }
        /* A16: stable compaction of exited particles (BASELINE config 5) */
        if (c->compact) {
            uint64_t o = 0;
            for (uint64_t i = 0; i < s->n; ++i) {
                if (s->status[i] != 0) continue;
                if (o != i) {
                    s->x[o] = s->x[i]; s->y[o] = s->y[i]; s->z[o] = s->z[i];
                    s->pid[o] = s->pid[i]; s->status[o] = 0; s->fragile[o] = s->fragile[i];
                    for (int k = 0; k < c->K; ++k) s->m[k][o] = s->m[k][i];
                }
                ++o;
            }
            s->n = o;
        }
        s->step = n + 1;
        if (c->bin_every > 0 && s->step % (uint64_t)c->bin_every == 0) {
            orc_bin_now(s);
            /* PAPER.md L108 / Fig. 2b (L218) "time integrated dosage": the gridded activity concentration of every
             * n-th step times the interval it stands for, summed (rectangle rule at the binning cadence) */
            if (s->dose) {
                size_t nc = (size_t)cg->nx * cg->ny * cg->nz * c->K;
                double V = cg->dx * cg->dy * cg->dz, T = (double)c->bin_every * c->dt;
                for (size_t i = 0; i < nc; ++i) s->dose[i] += s->conc_sum[i] / V * T;
            }
        }
    }
    return 0;
}

/* start accumulating the time-integrated concentration at every cadence binning from now on */
void orc_enable_dose(orc_sim *s)
{
    const orc_grid *g = &s->cfg.cgrid;
    if (!s->dose) s->dose = calloc((size_t)g->nx * g->ny * g->nz * s->cfg.K, sizeof(double));
    if (!s->dose) abort();
}

void orc_dose(const orc_sim *s, double *out)
{
    const orc_grid *g = &s->cfg.cgrid;
    size_t n = (size_t)g->nx * g->ny * g->nz * s->cfg.K;
    for (size_t i = 0; i < n; ++i) out[i] = s->dose ? s->dose[i] : 0.0;
}

/* ------------------------------------------------------------------ accessors (test hooks) */
uint64_t orc_num_particles(const orc_sim *s) { return s->n; }
uint64_t orc_step_index(const orc_sim *s) { return s->step; }
uint64_t orc_num_fragile(const orc_sim *s) { return s->n_frag; }
void orc_get_fragile(const orc_sim *s, uint64_t *out) { memcpy(out, s->frag_pids, s->n_frag * sizeof(uint64_t)); }
float orc_p_dry(const orc_sim *s, int k) { return s->p_dry[k]; }
float orc_p_wet(const orc_sim *s, int k) { return s->p_wet[k]; }
float orc_sigma_h(const orc_sim *s) { return s->sigma_h; }

void orc_get_particles(const orc_sim *s, double *x, double *y, double *z, double *m0, double *m1,
                       uint64_t *pid, uint8_t *status)
{
    for (uint64_t i = 0; i < s->n; ++i) {
        if (x) x[i] = s->x[i];
        if (y) y[i] = s->y[i];
        if (z) z[i] = s->z[i];
        if (m0) m0[i] = s->m[0][i];
        if (m1 && s->cfg.K > 1) m1[i] = s->m[1][i];
        if (pid) pid[i] = s->pid[i];
        if (status) status[i] = s->status[i];
    }
}

/* replace the whole particle state (single-step parity from an identical state, T1; binning
 * fed identical positions).  Does not touch the ledger. */
void orc_set_particles(orc_sim *s, uint64_t n, const double *x, const double *y, const double *z,
                       const double *m0, const double *m1, const uint64_t *pid, const uint8_t *status)
{
    grow(s, n);
    s->n = n;
    for (uint64_t i = 0; i < n; ++i) {
        s->x[i] = x[i]; s->y[i] = y[i]; s->z[i] = z[i];
        s->m[0][i] = m0[i];
        if (s->cfg.K > 1) s->m[1][i] = m1[i];
        s->pid[i] = pid ? pid[i] : i;
        s->status[i] = status ? status[i] : 0;
        s->fragile[i] = 0;
    }
}

void orc_set_step_index(orc_sim *s, uint64_t step) { s->step = step; }

void orc_ledger(const orc_sim *s, double *out /* [K][7] */)
{
    for (int k = 0; k < s->cfg.K; ++k) {
        double air = 0.0;
        for (uint64_t i = 0; i < s->n; ++i) if (s->status[i] == 0) air += s->m[k][i];
        for (int q = 0; q < ORC_NLEDGER; ++q) out[k * ORC_NLEDGER + q] = s->ledger[k][q];
        out[k * ORC_NLEDGER + 1] = air;
    }
}

/* concentration [K][nz][ny][nx] in Bq m^-3 = summed activity / cell volume (R10) */
void orc_concentration(const orc_sim *s, double *out)
{
    const orc_grid *g = &s->cfg.cgrid;
    size_t n = (size_t)g->nx * g->ny * g->nz * s->cfg.K;
    double V = g->dx * g->dy * g->dz;
    for (size_t i = 0; i < n; ++i) out[i] = s->conc_sum[i] / V;
}

void orc_counts(const orc_sim *s, uint32_t *out)
{
    const orc_grid *g = &s->cfg.cgrid;
    memcpy(out, s->cnt, (size_t)g->nx * g->ny * g->nz * sizeof(uint32_t));
}

/* deposition [K][ny][nx] in Bq m^-2; slack = the part of it carried by increments that lay
 * within face_delta of a cell face (could legitimately land in the neighbour cell) */
void orc_deposition(const orc_sim *s, double *out, double *slack)
{
    const orc_grid *g = &s->cfg.cgrid;
    size_t n = (size_t)g->nx * g->ny * s->cfg.K;
    double A = g->dx * g->dy;
    for (size_t i = 0; i < n; ++i) {
        out[i] = s->dep[i] / A;
        if (slack) slack[i] = s->dep_slack[i] / A;
    }
}

/* R13: from now on also keep the deposition map whose content decays on the ground.  Call before the first deposit
 * (it starts from the undecayed map as it stands, which is only right while that map is empty or freshly deposited). */
void orc_enable_ground_decay(orc_sim *s)
{
    const orc_grid *g = &s->cfg.cgrid;
    size_t n = (size_t)g->nx * g->ny * s->cfg.K;
    if (s->ground) return;
    s->ground = malloc(n * sizeof(double));
    s->ground_slack = malloc(n * sizeof(double));
    if (!s->ground || !s->ground_slack) abort();
    memcpy(s->ground, s->dep, n * sizeof(double));
    memcpy(s->ground_slack, s->dep_slack, n * sizeof(double));
}

/* the ground-decayed deposition [K][ny][nx] in Bq m^-2 at the current time, and its face slack */
void orc_deposition_ground(const orc_sim *s, double *out, double *slack)
{
    const orc_grid *g = &s->cfg.cgrid;
    size_t n = (size_t)g->nx * g->ny * s->cfg.K;
    double A = g->dx * g->dy;
    for (size_t i = 0; i < n; ++i) {
        out[i] = s->ground ? s->ground[i] / A : 0.0;
        if (slack) slack[i] = s->ground_slack ? s->ground_slack[i] / A : 0.0;
    }
}

uint64_t orc_injected(const orc_sim *s, uint64_t step) { return step < s->inj_cap ? s->inj_log[step] : 0; }

int32_t orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
void orc_set_num_threads(int32_t n)
{
#ifdef _OPENMP
    omp_set_num_threads(n);
#else
    (void)n;
#endif
}
