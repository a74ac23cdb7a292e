// lpm_api.cu — host side of the C ABI declared in include/lpm.h: handle, workspace carving,
// release schedule (R9), per-step scalar tables (R4 time weights, R8 decay scale), launch loop.
// No step of the path runs on the host: the host only computes scalars and enqueues kernels.
#include <math.h>
#include <stdio.h>
#include <string.h>

#include <mutex>
#include <new>
#include <vector>

#include "lpm_internal.h"

using namespace lpm;

namespace {

constexpr uint64_t kAlign = 256;
constexpr uint64_t kInjLog = 1u << 16;  // ring of per-step injected counts (compact mode)

struct Release {
    lpm_source src;
    double emit[LPM_MAX_NUCLIDES];
    uint64_t N, c, pid_offset, pid_stride;
    int64_t s_start, S;
    uint64_t base, n_local;
    bool fixed;  // installed by lpm_set_particles: every slot already born
};

struct Layout {
    uint64_t xyzq, q1, pid, cnt, conc, dep, ledger, air, ctrl, tile, injlog, stage, pair, blend, keys, perm, hist, partial, alt_xyzq, alt_q1, alt_pid, dose, mask, surf, total;
};

uint64_t up(uint64_t v) { return (v + kAlign - 1) / kAlign * kAlign; }

Layout make_layout(const lpm_grid &g, const lpm_meteo &met, uint64_t cap, int K, bool compact, bool sort, bool dose, bool zpair)
{
    Layout L{};
    const uint64_t cells3 = (uint64_t)g.nx * g.ny * g.nz, cells2 = (uint64_t)g.nx * g.ny;
    uint64_t o = 0;
    L.xyzq = o; o += up(16 * cap);
    L.q1 = o; o += K > 1 ? up(4 * cap) : 0;
    L.pid = o; o += compact ? up(4 * cap) : 0;
    L.cnt = o; o += up(4 * cells3);
    L.conc = o; o += up(8 * cells3 * K);
    L.dep = o; o += up(8 * cells2 * K);
    L.ledger = o; o += up(8 * 8 * LPM_MAX_NUCLIDES);
    L.air = o; o += up(8 * 2);
    L.ctrl = o; o += up(8 * 32);
    L.tile = o; o += compact ? up(8 * (cap / kScanTile + 2)) : 0;
    L.injlog = o; o += compact ? up(8 * kInjLog) : 0;
    L.stage = o; o += up(4 * cells3 * K);  // fp32 read-out staging for the *_host entry points
    L.pair = o; o += met.nt > 1 ? up(32ull * met.grid.nx * met.grid.ny * met.grid.nz) : 0;  // (F_s, F_s+1) per met cell
    const uint64_t mcells = (uint64_t)met.grid.nx * met.grid.ny * met.grid.nz;
    L.blend = o; o += up((zpair ? 32ull : 16ull) * mcells * (met.nt > 1 ? kBlendDepth : 1) + 32);  // z-fastest F(t_n), one buffer per fused step (+ 1 pad texel)
    L.keys = o; o += sort ? up(4 * cap) : 0;            // gather-locality pass: met-cell key per slot
    L.perm = o; o += sort && !compact ? 2 * up(4 * cap) : 0;  //   slots in met-cell order (slot-addressed store): current list + the one being built
    L.hist = o; o += sort ? up(4 * (mcells + 1)) : 0;   //   per-cell counts / offsets
    L.partial = o; o += sort ? up(4 * sort_partial_entries(mcells)) : 0;
    L.alt_xyzq = o; o += sort && compact ? up(16 * cap) : 0;           //   compact store: the records themselves are sorted,
    L.alt_q1 = o; o += sort && compact && K > 1 ? up(4 * cap) : 0;     //   through these alternate buffers
    L.alt_pid = o; o += sort && compact ? up(4 * cap) : 0;
    L.mask = o; o += up((uint64_t)((met.grid.nx + kMaskTile - 1) / kMaskTile) * ((met.grid.ny + kMaskTile - 1) / kMaskTile));  // plume mask tiles
    L.surf = o; o += met.kz_mode == 1 ? up(16ull * met.grid.nx * met.grid.ny * (met.nt > 1 ? kBlendDepth : 1)) : 0;  // R12 2-D fields per fused step
    L.dose = o; o += dose ? up(8 * cells3 * K) : 0;                    // time-integrated concentration (S 8(f)3)
    L.total = o;
    return L;
}

// zfast: strides of the library's z-fastest met buffers; otherwise x-fastest (only nx, ny, nz, the
// corner and the inverse spacings matter for the binning grid)
GridF gridf(const lpm_grid &g, bool zfast = false, const float *levels = nullptr)
{
    GridF f;
    memset(&f, 0, sizeof(f));
    if (levels) {
        f.nlev = g.nz;
        for (int k = 0; k < g.nz && k < kMaxLevels; ++k) f.zlev[k] = levels[k];
    }
    f.nx = g.nx; f.ny = g.ny; f.nz = g.nz;
    f.x0 = (float)g.x0; f.y0 = (float)g.y0; f.z0 = (float)g.z0;
    f.inv_dx = (float)(1.0 / g.dx); f.inv_dy = (float)(1.0 / g.dy); f.inv_dz = (float)(1.0 / g.dz);
    f.cx = (float)(-g.x0 / g.dx - 0.5); f.cy = (float)(-g.y0 / g.dy - 0.5); f.cz = (float)(-g.z0 / g.dz - 0.5);
    f.fx1 = (float)(g.nx - 1); f.fy1 = (float)(g.ny - 1); f.fz1 = (float)(g.nz - 1);
    f.ix2 = g.nx > 2 ? g.nx - 2 : 0; f.iy2 = g.ny > 2 ? g.ny - 2 : 0; f.iz2 = g.nz > 2 ? g.nz - 2 : 0;
    if (zfast) { f.ez = 1u; f.ex = (uint32_t)g.nz; f.ey = (uint32_t)g.nz * (uint32_t)g.nx; }
    else { f.ex = 1u; f.ey = (uint32_t)g.nx; f.ez = (uint32_t)g.nx * (uint32_t)g.ny; }
    f.sx = g.nx > 1 ? f.ex : 0u; f.sy = g.ny > 1 ? f.ey : 0u; f.sz = g.nz > 1 ? f.ez : 0u;
    return f;
}

// the gather-locality pass: a list of slot indices for the slot-addressed store, a physical sort of the
// records for the compact store (from 65536 slots of capacity, or when asked for)
constexpr uint64_t kSortAutoMin = 65536;
bool sort_enabled(const lpm_params *p)
{
    if (p->compact) return p->gather_sort > 0 || (p->gather_sort == 0 && p->capacity >= kSortAutoMin);
    return p->gather_sort >= 0;
}

// B8: z-pair texels in the blended buffers.  The physics they are instantiated for, and the auto rule.
constexpr uint64_t kPairAutoRatio = 16;
bool zpair_possible(const lpm_meteo *met, const lpm_params *p)
{
    return !p->compact && met->nt > 1 && p->dep_mode == 0 && met->kz_mode == 0 && met->z_levels_host == nullptr && p->drift == 0;
}
bool zpair_enabled(const lpm_meteo *met, const lpm_params *p)
{
    if (p->texel_pairs < 0 || !zpair_possible(met, p)) return false;
    if (p->texel_pairs > 0) return true;
    return p->capacity >= kPairAutoRatio * (uint64_t)met->grid.nx * met->grid.ny * met->grid.nz;
}

bool grid_ok(const lpm_grid *g)
{
    return g && g->nx > 0 && g->ny > 0 && g->nz > 0 && g->dx > 0 && g->dy > 0 && g->dz > 0 &&
           (uint64_t)g->nx * g->ny * g->nz < (1ull << 31);
}

// The step kernel addresses the time-blended met buffers with ONE 32-bit texel index that includes the buffer
// (lpm_step.cu, step_once: c.o += e.buf * snap_cells, e.buf < kBlendDepth): with more than one snapshot all kBlendDepth
// buffers together must stay below 2^32 texels, i.e. the met grid below 2^28 cells (a single snapshot has one buffer).
bool met_index_ok(const lpm_meteo *met)
{
    const uint64_t cells = (uint64_t)met->grid.nx * met->grid.ny * met->grid.nz;
    return met->nt <= 1 || (uint64_t)kBlendDepth * cells < (1ull << 32);
}

}  // namespace

struct lpm_handle {
    lpm_grid cg;
    lpm_meteo met;
    lpm_nuclide nuc[LPM_MAX_NUCLIDES];
    lpm_params prm;
    bool has_levels;
    bool zpair;   // B8: the blended buffers hold 32-byte z-pair texels
    int perm_cur; // which half of L.perm holds the current slot list
    bool sort_by_slot;  // fused sort keys indexed by slot (large ensembles), else by list position
    int sort_period;    // model steps between two gather sorts when gather_sort = 0 (auto)
    float zlev[kMaxLevels];   // non-uniform level heights (fp32 parameters), copied from meteo.z_levels_host
    int K;
    cudaStream_t st;
    char *ws;
    Layout L;
    // derived constants (R5, R8)
    float sigma_h, p_dry[LPM_MAX_NUCLIDES], p_wet[LPM_MAX_NUCLIDES];
    double f_decay[LPM_MAX_NUCLIDES], ln_rho[LPM_MAX_NUCLIDES], dec_scale[LPM_MAX_NUCLIDES], wet_scale[LPM_MAX_NUCLIDES];
    int dry_mode;
    bool rain_on;
    double rx0, rx1, ry0, ry1, rt0, rt1;
    std::vector<Release> rel;
    uint64_t next_base;
    uint64_t step, bin_step;
    int pair_snap;  // snapshot index s whose pair (s, s+1) the pair buffer holds, -1 = none
    // a0: the blend buffers hold F(t_n) for steps [blend_step0, blend_step0 + blend_n) (blend_n = 0: nothing)
    uint64_t blend_step0;
    int blend_n;
    // gather-locality pass: the perm buffer lists slots [0, perm_n) of the (single) release as sorted at step perm_step
    uint64_t perm_n, perm_step;
    bool perm_valid;
    // keys + histogram of slots [0, keys_n) left by the step launch that ended at step keys_step
    uint64_t keys_n, keys_step;
    bool keys_ready;
    uint64_t csort_step;  // compact store: step of the last physical sort
    bool bbox_valid;      // the mask tiles hold the met columns of the particles as the last step launch left them
    double dep_bound[LPM_MAX_NUCLIDES];  // largest activity a particle can carry (fixed-point scale of the deposit tables)
    double lam_dt[LPM_MAX_NUCLIDES];     // lambda_k dt
    uint64_t dep_ref[LPM_MAX_NUCLIDES];  // R13 (ground_decay): the map of nuclide k holds activity referred to this step's time
    bool binned;
    int sms, occ;
    uint64_t launches;
    // timing hooks: event pairs around step / binning launches
    bool timing;
    struct Span { cudaEvent_t a, b; int kind; bool pre; double units; };   // pre: the step launch right before one with the binning epilogue
    std::vector<Span> spans;
    std::vector<cudaEvent_t> ev_pool;
    double t_ms[5], t_units[5];   // kinds: 0 step launches, 1 binning (memset + stand-alone kernel), 2 sorts, 3 step launches with the fused
                                  // binning epilogue (also counted in 0), 4 the step launches right before those (also in 0)
    int last_step_span;           // index into spans of the latest kind-0 span, -1 = none
    uint64_t t_base, t_base_bin;  // device counters (particle-steps executed, particles binned) at lpm_set_timing
    uint64_t t_launches[5];
    int sticky;
    char err[512];
};

namespace {

int fail(lpm_handle *h, int code, const char *msg)
{
    if (h) snprintf(h->err, sizeof(h->err), "%s", msg);
    return code;
}

int cuda_fail(lpm_handle *h, cudaError_t e, const char *where)
{
    if (h) {
        snprintf(h->err, sizeof(h->err), "%s: %s", where, cudaGetErrorString(e));
        h->sticky = LPM_ERR_CUDA;
    }
    return LPM_ERR_CUDA;
}

#define CK(call)                                                   \
    do {                                                           \
        cudaError_t e_ = (call);                                   \
        if (e_ != cudaSuccess) return cuda_fail(h, e_, #call);     \
    } while (0)

cudaEvent_t ev_get(lpm_handle *h)
{
    if (!h->ev_pool.empty()) { cudaEvent_t e = h->ev_pool.back(); h->ev_pool.pop_back(); return e; }
    cudaEvent_t e = nullptr;
    if (cudaEventCreate(&e) != cudaSuccess) return nullptr;
    return e;
}

// open / close a timed span of kind 0 (step kernel) or 1 (binning) on the handle's stream
int span_open(lpm_handle *h, int kind, double units)
{
    if (!h->timing) return -1;
    lpm_handle::Span sp{ev_get(h), ev_get(h), kind, false, units};
    if (!sp.a || !sp.b) {   // no event to be had: this launch goes untimed (its units are not counted either)
        if (sp.a) h->ev_pool.push_back(sp.a);
        if (sp.b) h->ev_pool.push_back(sp.b);
        return -1;
    }
    cudaEventRecord(sp.a, h->st);
    if (kind == 3 && h->last_step_span >= 0 && h->last_step_span < (int)h->spans.size()) h->spans[h->last_step_span].pre = true;
    h->spans.push_back(sp);
    h->t_units[kind] += units;
    h->t_launches[kind]++;
    if (kind == 3) { h->t_units[0] += units; h->t_launches[0]++; }
    if (kind == 0) h->last_step_span = (int)h->spans.size() - 1;   // (sort and memset spans in between do not matter)
    if (kind == 3) h->last_step_span = -1;
    return (int)h->spans.size() - 1;
}
void span_close(lpm_handle *h, int id)
{
    if (id >= 0) cudaEventRecord(h->spans[id].b, h->st);
}
void spans_collect(lpm_handle *h)
{
    for (auto &sp : h->spans) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, sp.a, sp.b) == cudaSuccess) {
            h->t_ms[sp.kind] += (double)ms;
            if (sp.kind == 3) h->t_ms[0] += (double)ms;
            if (sp.pre) { h->t_ms[4] += (double)ms; h->t_launches[4]++; h->t_units[4] += sp.units; }
        }
        h->ev_pool.push_back(sp.a);
        h->ev_pool.push_back(sp.b);
    }
    h->spans.clear();
    h->last_step_span = -1;
}

double G_of(const lpm_handle *h, int k, uint64_t step) { return exp((double)step * h->ln_rho[k]); }

// R9: local particles of release r born at steps <= step
uint64_t born_local(const Release &r, int64_t step)
{
    if (r.fixed) return r.n_local;
    const int64_t rs = step - r.s_start;
    if (rs < 0) return 0;
    if (r.N > 0) {
        uint64_t B = r.N;
        if (rs + 1 < r.S) {
            const unsigned __int128 num = (unsigned __int128)(uint64_t)(rs + 1) * r.N;
            B = (uint64_t)((num + (uint64_t)r.S - 1) / (uint64_t)r.S);
            if (B > r.N) B = r.N;
        }
        if (B <= r.pid_offset) return 0;
        return (B - r.pid_offset + r.pid_stride - 1) / r.pid_stride;
    }
    const int64_t steps = rs + 1 < r.S ? rs + 1 : r.S;
    return r.c * (uint64_t)steps;
}

void fill_entry(const lpm_handle *h, uint64_t n, StepEntry &e)
{
    const double t = (double)n * h->prm.dt;
    int s = 0;
    float a = 0.0f;
    if (h->met.nt > 1) {  // R4 time weight, fp32-rounded parameter
        double r = floor((t - h->met.t0) / h->met.dt_snap);
        if (r < 0.0) r = 0.0;
        if (r > (double)(h->met.nt - 2)) r = (double)(h->met.nt - 2);
        s = (int)r;
        double ad = (t - (h->met.t0 + (double)s * h->met.dt_snap)) / h->met.dt_snap;
        if (ad < 0.0) ad = 0.0;
        if (ad > 1.0) ad = 1.0;
        a = (float)ad;
    }
    const bool raining = h->rain_on && t >= h->rt0 && t < h->rt1;  // G6
    e.a = a;
    e.buf = 0;
    e.pad_ = 0;
    e.snap = s | (raining ? 1 << 16 : 0);
    for (int k = 0; k < LPM_MAX_NUCLIDES; ++k) {
        e.G[k] = k < h->K ? G_of(h, k, n) : 1.0;
        e.Gf[k] = (float)e.G[k];
        e.Gp[k] = k < h->K ? (float)(e.G[k] * (double)h->p_dry[k]) : 0.0f;
        e.Gps[k] = 0.0f;
    }
}

void base_args(const lpm_handle *h, StepArgs &A)
{
    memset(&A, 0, sizeof(A));
    A.xyzq = (float4 *)(h->ws + h->L.xyzq);
    A.q1 = h->K > 1 ? (float *)(h->ws + h->L.q1) : nullptr;
    A.pid = h->prm.compact ? (uint32_t *)(h->ws + h->L.pid) : nullptr;
    A.blend = (const float4 *)(h->ws + h->L.blend);
    A.zpair = h->zpair ? 1 : 0;
    const lpm_grid &mg = h->met.grid;
    A.snap_cells = (uint64_t)mg.nx * mg.ny * mg.nz;
    A.mg = gridf(mg, true, h->has_levels ? h->zlev : nullptr);
    A.bx0 = (float)mg.x0; A.bx1 = (float)(mg.x0 + mg.nx * mg.dx);
    A.by0 = (float)mg.y0; A.by1 = (float)(mg.y0 + mg.ny * mg.dy);
    A.cg = gridf(h->cg);
    A.dep = (double *)(h->ws + h->L.dep);
    A.dep_stride = (uint64_t)h->cg.nx * h->cg.ny;
    A.bern = h->prm.dep_mode == 1 ? 1 : 0;
    A.eq3 = h->met.kz_mode == 1 ? 1 : 0;
    A.drift = h->prm.drift == 1 ? 1 : 0;
    A.surf = A.eq3 ? (const float4 *)(h->ws + h->L.surf) : nullptr;
    A.any_dep = (!A.bern && (h->dry_mode != kDryNone || h->rain_on)) ? 1 : 0;
    for (int w = 0; w < 2 * LPM_MAX_NUCLIDES; ++w) {
        // S = largest power of two <= 2^20 / (largest possible increment): activity <= dep_bound, one step
        // deposits at most the fraction p_dry (dry) or p_wet (wet) of it.  Only efficiency depends on the
        // bound: an increment outside [2^17, 2^20) / S takes the direct fp64 RED.
        const int k = w / 2;
        const double frac = k < h->K ? (w & 1 ? (double)h->p_wet[k] : (double)h->p_dry[k]) : 0.0;
        // (ground decay: the increments of a launch grow by up to exp(lambda dt kMaxFused) relative to its first step)
        const double grow = h->prm.ground_decay && k < h->K ? exp(h->lam_dt[k] * kMaxFused) : 1.0;
        const double inc_max = (k < h->K ? h->dep_bound[k] : 0.0) * frac * grow;
        int e = 0;
        if (inc_max > 0.0) { frexp(1048576.0 / inc_max, &e); e -= 1; }
        if (e > 100) e = 100;
        if (e < -100) e = -100;
        A.dep_scale[w] = (float)ldexp(1.0, e);
        A.dep_inv_scale[w] = ldexp(1.0, -e);
    }
    A.dt = (float)h->prm.dt;
    A.sigma_h = h->sigma_h;
    A.kz_min = (float)h->met.kz_min;
    A.H = (float)h->met.H_mix;
    A.h_dep = (float)h->prm.h_dep;
    A.dry_mode = h->dry_mode;
    A.absorb = h->prm.boundary_mode == LPM_BOUNDARY_ABSORB;
    for (int k = 0; k < LPM_MAX_NUCLIDES; ++k) {
        A.p_dry[k] = h->p_dry[k]; A.p_wet[k] = h->p_wet[k];
        A.dec_scale[k] = h->dec_scale[k]; A.wet_scale[k] = h->wet_scale[k];
        A.wet_scale_f[k] = (float)h->wet_scale[k];
    }
    A.rx0 = (float)h->rx0; A.rx1 = (float)h->rx1; A.ry0 = (float)h->ry0; A.ry1 = (float)h->ry1;
    A.seed_lo = (uint32_t)h->prm.seed; A.seed_hi = (uint32_t)(h->prm.seed >> 32);
    for (uint32_t r = 0; r < 10; ++r) {  // R1 key schedule: the key is bumped by the Weyl constants between rounds
        A.rk[2 * r] = A.seed_lo + r * 0x9E3779B9u;
        A.rk[2 * r + 1] = A.seed_hi + r * 0xBB67AE85u;
    }
    A.ledger = (double *)(h->ws + h->L.ledger);
    A.ctrl = (uint64_t *)(h->ws + h->L.ctrl);
    A.tile_state = h->prm.compact ? (uint64_t *)(h->ws + h->L.tile) : nullptr;
}

int grid_blocks(const lpm_handle *h, uint64_t n)
{
    const uint64_t want = (n + kStepThreads - 1) / kStepThreads;
    const uint64_t maxb = (uint64_t)h->sms * (uint64_t)(h->occ > 0 ? h->occ : 1);
    return (int)(want < maxb ? (want ? want : 1) : maxb);
}

// control block (uint64 words of L.ctrl): [0..2] compact store counts, [3] particle-steps executed (cumulative),
// [4..6] hole list / fill counters, [8..15] per-release emitted counts (compact), [16] tile ticket of the slot kernel,
// [17], [18] live length of the slot list in half 0 / 1 of L.perm, [19] particles binned (cumulative),
// [20] cells that held a particle at the last lpm_touched_cells, [22] |u|max, |v|max of the met interval
constexpr int kCtrlSteps = 3, kCtrlLive = 17, kCtrlBinned = 19, kCtrlTouched = 20;

uint32_t *perm_half(const lpm_handle *h, int half) { return (uint32_t *)(h->ws + h->L.perm) + (uint64_t)half * (up(4 * h->prm.capacity) / 4); }

// fixed-point scale of the CTA-private concentration sums: largest power of two S with q_max S < 2^20, where the
// largest stored q is bounded by dep_bound / G(now) (q = activity / G(t), and a particle never gains activity)
void bin_scales(const lpm_handle *h, uint64_t step, float *scale, double *inv_scale)
{
    for (int k = 0; k < LPM_MAX_NUCLIDES; ++k) {
        const double qmax = k < h->K ? h->dep_bound[k] / G_of(h, k, step) : 0.0;
        int e = 0;
        if (qmax > 0.0) { frexp(1048576.0 / qmax, &e); e -= 1; }
        if (e > 100) e = 100;
        if (e < -100) e = -100;
        scale[k] = (float)ldexp(1.0, e);
        inv_scale[k] = ldexp(1.0, -e);
    }
}

int do_bin(lpm_handle *h)
{
    const uint64_t cells3 = (uint64_t)h->cg.nx * h->cg.ny * h->cg.nz;
    const int span = span_open(h, 1, 0.0);
    // the count grid and the K sum grids lie back to back in the workspace: one memset
    CK(cudaMemsetAsync(h->ws + h->L.cnt, 0, (h->L.conc - h->L.cnt) + 8 * cells3 * h->K, h->st));
    BinArgs B{};
    B.q1 = h->K > 1 ? (const float *)(h->ws + h->L.q1) : nullptr;
    B.cg = gridf(h->cg);
    B.cnt = (uint32_t *)(h->ws + h->L.cnt);
    B.conc = (double *)(h->ws + h->L.conc);
    B.cells3 = cells3;
    B.K = h->K;
    B.n_binned = (uint64_t *)(h->ws + h->L.ctrl) + kCtrlBinned;
    bin_scales(h, h->step, B.scale, B.inv_scale);
    const int max_blocks = h->sms * 8;
    if (h->prm.compact) {
        B.xyzq = (const float4 *)(h->ws + h->L.xyzq);
        B.n_dev = (const uint64_t *)(h->ws + h->L.ctrl) + 2;
        CK(launch_bin(B, max_blocks, h->st));
        h->launches++;
    } else {
        for (const Release &r : h->rel) {
            const uint64_t n = born_local(r, (int64_t)h->step - 1);
            if (!n) continue;
            B.xyzq = (const float4 *)(h->ws + h->L.xyzq) + r.base;
            if (B.q1) B.q1 = (const float *)(h->ws + h->L.q1) + r.base;
            B.n = n;
            const uint64_t want = (n + 1023) / 1024;
            CK(launch_bin(B, (int)(want < (uint64_t)max_blocks ? want : (uint64_t)max_blocks), h->st));
            h->launches++;
        }
    }
    span_close(h, span);
    h->bin_step = h->step;
    h->binned = true;
    return LPM_OK;
}

// a0: make the blend buffers hold F(t_n) for the m steps starting at h->step (entries A.tab[0..m)
// are filled and lie inside one met interval) and point the entries at them.
int ensure_blend(lpm_handle *h, StepArgs &A, int m, int m_max)
{
    const lpm_grid &g = h->met.grid;
    const float4 *met = (const float4 *)h->met.fields_dev;
    float4 *blend = (float4 *)(h->ws + h->L.blend);
    if (h->met.nt == 1) {
        if (h->blend_n == 0) {
            CK(launch_transpose(met, blend, g.nx, g.ny, g.nz, h->st));
            h->launches++;
            if (h->met.kz_mode == 1) {  // R12: the single snapshot of the 2-D fields, as it is
                const float a0 = 0.0f;
                CK(launch_blend_surface((const float4 *)h->met.surface_dev, (const float4 *)h->met.surface_dev, (float4 *)(h->ws + h->L.surf),
                                        (uint64_t)g.nx * g.ny, 1, &a0, h->st));
                h->launches++;
            }
            h->blend_n = 1;
        }
        for (int s = 0; s < m; ++s) A.tab[s].buf = 0;
        return LPM_OK;
    }
    const int sn = A.tab[0].snap & 0xffff;
    if (sn != h->pair_snap) {
        CK(launch_pair_repack(met + (uint64_t)sn * A.snap_cells, met + (uint64_t)(sn + 1) * A.snap_cells, h->ws + h->L.pair,
                              g.nx, g.ny, g.nz, (uint32_t *)(A.ctrl + 22), h->st));
        h->launches++;
        h->pair_snap = sn;
        h->blend_n = 0;
    }
    if (!(h->blend_n > 0 && h->step >= h->blend_step0 && h->step + (uint64_t)m <= h->blend_step0 + (uint64_t)h->blend_n)) {
        float a[kBlendDepth];
        int cnt = 0;
        for (; cnt < m; ++cnt) a[cnt] = A.tab[cnt].a;
        if (m_max < kBlendDepth) {  // short launches (compact mode, steps_per_launch): blend ahead, reuse over the next launches
            for (; cnt < kBlendDepth; ++cnt) {
                StepEntry e;
                fill_entry(h, h->step + (uint64_t)cnt, e);
                if ((e.snap & 0xffff) != sn) break;
                a[cnt] = e.a;
            }
        }
        // plume box: columns reachable within the cnt steps these buffers serve (B6)
        BlendBox box{};
        box.flags = h->bbox_valid ? (const uint8_t *)(h->ws + h->L.mask) : nullptr;
        box.uvmax = (const uint32_t *)(A.ctrl + 22);
        box.nx = g.nx; box.ny = g.ny; box.nz = g.nz;
        const double walk = 5.768 * (double)h->sigma_h * 1.0001;
        box.reach_x = (float)((double)cnt * h->prm.dt / g.dx * 1.0001); box.reach_y = (float)((double)cnt * h->prm.dt / g.dy * 1.0001);
        box.walk_x = (float)((double)cnt * walk / g.dx); box.walk_y = (float)((double)cnt * walk / g.dy);
        for (const Release &r : h->rel) {
            if (r.fixed || box.n_src >= LPM_MAX_RELEASES) continue;
            int si = (int)floor((r.src.x - g.x0) / g.dx), sj = (int)floor((r.src.y - g.y0) / g.dy);
            box.src_i[box.n_src] = si < 0 ? 0 : (si > g.nx - 1 ? g.nx - 1 : si);
            box.src_j[box.n_src] = sj < 0 ? 0 : (sj > g.ny - 1 ? g.ny - 1 : sj);
            box.n_src++;
        }
        CK(launch_blend(h->ws + h->L.pair, blend, A.snap_cells, cnt, a, &box, h->zpair, h->st));
        h->launches++;
        if (h->met.kz_mode == 1) {  // R12: the 2-D fields (u*, 1/L, Hz) of the same steps
            const uint64_t c2 = (uint64_t)g.nx * g.ny;
            const float4 *sf = (const float4 *)h->met.surface_dev;
            CK(launch_blend_surface(sf + (uint64_t)sn * c2, sf + (uint64_t)(sn + 1) * c2, (float4 *)(h->ws + h->L.surf), c2, cnt, a, h->st));
            h->launches++;
        }
        h->blend_step0 = h->step;
        h->blend_n = cnt;
    }
    for (int s = 0; s < m; ++s) A.tab[s].buf = (uint32_t)(h->step + (uint64_t)s - h->blend_step0);
    return LPM_OK;
}

}  // namespace

extern "C" {

int32_t lpm_version(void) { return 100; }

const char *lpm_status_string(int32_t s)
{
    switch (s) {
        case LPM_OK: return "ok";
        case LPM_ERR_INVALID_ARG: return "invalid argument";
        case LPM_ERR_NO_DEVICE: return "no sm_100 CUDA device (there is no CPU fallback)";
        case LPM_ERR_WORKSPACE_TOO_SMALL: return "workspace too small";
        case LPM_ERR_CAPACITY: return "release does not fit into the particle capacity";
        case LPM_ERR_STATE: return "call order";
        case LPM_ERR_CUDA: return "CUDA error";
        default: return "unknown status";
    }
}

int32_t lpm_workspace_bytes(const lpm_grid *g, const lpm_meteo *met, const lpm_params *p, int32_t K, uint64_t *bytes)
{
    if (!grid_ok(g) || !met || !grid_ok(&met->grid) || met->nt < 1 || !p || !bytes || K < 1 || K > LPM_MAX_NUCLIDES || p->capacity == 0 || p->capacity >= (1ull << 32))
        return LPM_ERR_INVALID_ARG;
    if (!met_index_ok(met)) return LPM_ERR_INVALID_ARG;
    *bytes = make_layout(*g, *met, p->capacity, K, p->compact != 0, sort_enabled(p), p->dose != 0, zpair_enabled(met, p)).total;
    return LPM_OK;
}

int32_t lpm_schedule_born(uint64_t N, uint64_t pid_offset, uint64_t pid_stride, int64_t s_start, int64_t S,
                          int64_t step, uint64_t *born)
{
    if (!born || N == 0 || pid_stride == 0 || S < 1) return LPM_ERR_INVALID_ARG;
    Release r{};
    r.N = N; r.pid_offset = pid_offset; r.pid_stride = pid_stride; r.s_start = s_start; r.S = S;
    *born = born_local(r, step);
    return LPM_OK;
}

int32_t lpm_create(const lpm_grid *cg, const lpm_meteo *met, const lpm_nuclide *nuc, int32_t K, const lpm_params *p,
                   void *ws, uint64_t ws_bytes, void *stream, lpm_handle **out)
{
    if (!out) return LPM_ERR_INVALID_ARG;
    *out = nullptr;
    if (!grid_ok(cg) || !met || !grid_ok(&met->grid) || !nuc || !p || !ws || K < 1 || K > LPM_MAX_NUCLIDES)
        return LPM_ERR_INVALID_ARG;
    if (met->kz_mode < 0 || met->kz_mode > 1 || (met->kz_mode == 1 && (!met->surface_dev || ((uintptr_t)met->surface_dev & 15)))) return LPM_ERR_INVALID_ARG;
    if (met->z_levels_host) {
        if (met->grid.nz > kMaxLevels) return LPM_ERR_INVALID_ARG;
        for (int k = 1; k < met->grid.nz; ++k) if (!(met->z_levels_host[k] > met->z_levels_host[k - 1])) return LPM_ERR_INVALID_ARG;
    }
    if (met->nt < 1 || met->nt > 32767 || !met->fields_dev || ((uintptr_t)met->fields_dev & 15) || ((uintptr_t)ws & 255))
        return LPM_ERR_INVALID_ARG;
    if (!met_index_ok(met)) return LPM_ERR_INVALID_ARG;
    if (!(p->dt > 0) || p->capacity == 0 || p->capacity >= (1ull << 32) || !(met->H_mix > 0) || met->Kh < 0 ||
        (met->nt > 1 && !(met->dt_snap > 0)) || p->bin_every < 0 || p->steps_per_launch < 0 || !(p->h_dep > 0) || p->dep_mode < 0 ||
        p->dep_mode > 1 || p->drift < 0 || p->drift > 1 || (p->drift == 1 && met->kz_mode == 1) || p->texel_pairs < -1 || p->texel_pairs > 1 || p->ground_decay < 0 || p->ground_decay > 1 ||
        (p->texel_pairs == 1 && !zpair_possible(met, p)))
        return LPM_ERR_INVALID_ARG;
    int ndev = 0, dev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return LPM_ERR_NO_DEVICE;
    // (attributes, not cudaGetDeviceProperties: that call takes milliseconds, and bench.py re-creates the handle at every wrap of a looped config)
    int cc_major = 0, n_sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&cc_major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&n_sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return LPM_ERR_NO_DEVICE;
    if (cc_major != 10) return LPM_ERR_NO_DEVICE;

    const Layout L = make_layout(*cg, *met, p->capacity, K, p->compact != 0, sort_enabled(p), p->dose != 0, zpair_enabled(met, p));
    if (ws_bytes < L.total) return LPM_ERR_WORKSPACE_TOO_SMALL;

    lpm_handle *h = new (std::nothrow) lpm_handle();
    if (!h) return LPM_ERR_INVALID_ARG;
    h->cg = *cg; h->met = *met; h->prm = *p; h->K = K;
    h->has_levels = met->z_levels_host != nullptr;
    h->zpair = zpair_enabled(met, p);
    if (h->has_levels) for (int k = 0; k < met->grid.nz; ++k) h->zlev[k] = (float)met->z_levels_host[k];
    h->met.z_levels_host = nullptr;  // copied: the caller's array is not needed after lpm_create
    for (int k = 0; k < K; ++k) h->nuc[k] = nuc[k];
    h->st = (cudaStream_t)stream;
    h->ws = (char *)ws;
    h->L = L;
    h->sms = n_sms;
    h->err[0] = 0;
    h->pair_snap = -1;
    h->last_step_span = -1;
    // R5 / R8 constants: double formula, rounded once to fp32 where the kernels consume fp32
    h->sigma_h = (float)sqrt(2.0 * met->Kh * p->dt);
    {
        // Auto period of the gather sort: what un-sorts a warp is the horizontal random walk (advection moves neighbours
        // together), so the list is worth keeping for about as many steps as the walk needs to cross a met cell,
        // (dx / sigma_h)^2; measured optima 32 (c3: 31), 48-64 (c4: 62), 64 (c2: 250, c5: 100) -> 0.8 x that, in whole
        // launches of kMaxFused steps, between 32 and 64.
        const double dmin = met->grid.dx < met->grid.dy ? met->grid.dx : met->grid.dy;
        const double cross = h->sigma_h > 0.0f ? 0.8 * (dmin / h->sigma_h) * (dmin / h->sigma_h) : 1e9;
        int per = cross > 1e6 ? 64 : (int)(cross / kMaxFused + 0.5) * kMaxFused;
        h->sort_period = per < kSortPeriod ? kSortPeriod : (per > 2 * kSortPeriod ? 2 * kSortPeriod : per);
        // compact store: the record order also feeds the binning kernel's atomics (c5: 50 % of its roofline at 32, 45 % at 64)
        if (p->compact) h->sort_period = kSortPeriod;
    }
    // uniform dry deposition folds into the scalar G only in the expected-mass form; Bernoulli trials (R11) are per particle
    const bool eligible_everywhere = p->h_dep >= met->H_mix;
    const bool uniform = eligible_everywhere && p->dep_mode != 1;
    bool any_dry = false;
    for (int k = 0; k < K; ++k) {
        h->p_dry[k] = nuc[k].vd > 0 ? (float)(-expm1(-nuc[k].vd * p->dt / p->h_dep)) : 0.0f;
        h->p_wet[k] = nuc[k].lambda_wet > 0 ? (float)(-expm1(-nuc[k].lambda_wet * p->dt)) : 0.0f;
        any_dry |= h->p_dry[k] > 0.0f;
        const double lam_dt = nuc[k].half_life_s > 0 ? M_LN2 * p->dt / nuc[k].half_life_s : 0.0;
        h->f_decay[k] = exp(-lam_dt);
        h->lam_dt[k] = lam_dt;
        const double keep_dry = uniform ? 1.0 - (double)h->p_dry[k] : 1.0;
        h->ln_rho[k] = -lam_dt + (uniform ? log1p(-(double)h->p_dry[k]) : 0.0);
        h->dec_scale[k] = -expm1(-lam_dt) * keep_dry;
        h->wet_scale[k] = keep_dry * (double)h->p_wet[k];
    }
    h->dry_mode = !any_dry ? kDryNone : (eligible_everywhere ? kDryUniform : kDryLayer);
    // Scatter order of the gather sort.  Many particles per met cell AND per-step deposits through the CTA-private tables:
    // the slot-order scatter keeps each cell's slots ascending, i.e. sorted by age, and particles of one age sit together
    // (same map cell, neighbouring state records), which the step kernel gains more from than the scatter costs.  Otherwise
    // (Bernoulli deposition, no dry deposition, smaller ensembles) the cheaper list-order scatter.
    h->sort_by_slot = !p->compact && p->dep_mode == 0 && h->dry_mode != kDryNone &&
                      p->capacity >= kPairAutoRatio * (uint64_t)met->grid.nx * met->grid.ny * met->grid.nz;
    h->occ = step_max_blocks_per_sm(K, p->compact != 0, h->dry_mode, p->dep_mode == 1, met->kz_mode == 1, met->z_levels_host != nullptr || p->drift == 1, h->zpair);
    if (cudaMemsetAsync(ws, 0, L.total, h->st) != cudaSuccess) { delete h; return LPM_ERR_CUDA; }
    h->launches++;
    *out = h;
    return LPM_OK;
}

int32_t lpm_restart(lpm_handle *h)
{
    if (!h) return LPM_ERR_INVALID_ARG;
    if (h->sticky) return h->sticky;
    for (const Release &r : h->rel) if (r.fixed) return fail(h, LPM_ERR_STATE, "lpm_restart: the state was installed by lpm_set_particles, there is no release to start again");
    // everything that accumulates or counts; the particle store needs no clearing (a slot is initialised when its particle is born)
    const uint64_t cells3 = (uint64_t)h->cg.nx * h->cg.ny * h->cg.nz, cells2 = (uint64_t)h->cg.nx * h->cg.ny;
    const Layout &L = h->L;
    CK(cudaMemsetAsync(h->ws + L.cnt, 0, (L.conc - L.cnt) + 8 * cells3 * h->K, h->st));
    CK(cudaMemsetAsync(h->ws + L.dep, 0, 8 * cells2 * h->K, h->st));
    CK(cudaMemsetAsync(h->ws + L.ledger, 0, L.tile - L.ledger, h->st));    // ledger, airborne scratch, control block
    if (h->prm.compact) CK(cudaMemsetAsync(h->ws + L.tile, 0, L.stage - L.tile, h->st));   // look-back states, injected log
    if (h->prm.dose) CK(cudaMemsetAsync(h->ws + L.dose, 0, 8 * cells3 * h->K, h->st));
    h->launches += 4;
    h->step = 0; h->bin_step = 0; h->binned = false;
    h->t_base = 0; h->t_base_bin = 0;   // the device counters lpm_get_timing subtracts these from were zeroed with the control block
    h->pair_snap = -1; h->blend_n = 0; h->blend_step0 = 0; h->bbox_valid = false;
    h->perm_valid = false; h->perm_n = 0; h->perm_step = 0; h->perm_cur = 0; h->keys_ready = false; h->csort_step = 0;
    for (int k = 0; k < LPM_MAX_NUCLIDES; ++k) { h->dep_ref[k] = 0; h->dep_bound[k] = 0.0; }
    for (const Release &r : h->rel)
        for (int k = 0; k < h->K; ++k) if (r.emit[k] > h->dep_bound[k]) h->dep_bound[k] = r.emit[k];
    return LPM_OK;
}

int32_t lpm_destroy(lpm_handle *h)
{
    if (!h) return LPM_ERR_INVALID_ARG;
    cudaStreamSynchronize(h->st);
    spans_collect(h);
    for (cudaEvent_t e : h->ev_pool) cudaEventDestroy(e);
    delete h;
    return LPM_OK;
}

const char *lpm_last_error(lpm_handle *h) { return h ? h->err : "null handle"; }

int32_t lpm_set_rain(lpm_handle *h, double x0, double x1, double y0, double y1, double t0, double t1)
{
    if (!h || !(x1 > x0) || !(y1 > y0) || !(t1 > t0)) return fail(h, LPM_ERR_INVALID_ARG, "lpm_set_rain: empty box or interval");
    h->rain_on = true;
    h->rx0 = x0; h->rx1 = x1; h->ry0 = y0; h->ry1 = y1; h->rt0 = t0; h->rt1 = t1;
    return LPM_OK;
}

int32_t lpm_release(lpm_handle *h, const lpm_source *src, const double *act, uint64_t N, double rate, uint64_t off, uint64_t stride)
{
    if (!h || !src || !act || stride < 1) return fail(h, LPM_ERR_INVALID_ARG, "lpm_release: null or zero stride");
    if (h->rel.size() >= LPM_MAX_RELEASES) return fail(h, LPM_ERR_CAPACITY, "lpm_release: too many releases");
    Release r{};
    r.src = *src;
    r.s_start = (int64_t)ceil(src->t_start / h->prm.dt);
    r.S = (int64_t)ceil((src->t_end - src->t_start) / h->prm.dt);
    if (r.S < 1) r.S = 1;
    if ((int64_t)h->step > r.s_start) return fail(h, LPM_ERR_STATE, "lpm_release: release starts before the current step");
    r.pid_offset = off; r.pid_stride = stride;
    if (N > 0) {
        r.N = N;
        r.n_local = off < N ? (N - off + stride - 1) / stride : 0;
        for (int k = 0; k < h->K; ++k) r.emit[k] = act[k] / (double)N;
        if (off + (r.n_local ? r.n_local - 1 : 0) * stride >= (1ull << 32)) return fail(h, LPM_ERR_INVALID_ARG, "lpm_release: particle ids must stay below 2^32");
    } else {
        if (stride != 1) return fail(h, LPM_ERR_INVALID_ARG, "lpm_release: rate mode needs pid_stride 1");
        r.c = (uint64_t)llround(rate * h->prm.dt);
        if (r.c == 0) return fail(h, LPM_ERR_INVALID_ARG, "lpm_release: rate*dt rounds to zero");
        r.n_local = r.c * (uint64_t)r.S;
        for (int k = 0; k < h->K; ++k) r.emit[k] = act[k] / ((double)r.c * (double)r.S);
        if (off + r.n_local >= (1ull << 32)) return fail(h, LPM_ERR_INVALID_ARG, "lpm_release: particle ids must stay below 2^32");
    }
    if (!h->prm.compact) {
        for (const Release &o : h->rel) if (o.fixed) return fail(h, LPM_ERR_STATE, "lpm_release: state was replaced by lpm_set_particles");
        if (h->next_base + r.n_local > h->prm.capacity) return fail(h, LPM_ERR_CAPACITY, "lpm_release: particles exceed capacity");
        r.base = h->next_base;
        h->next_base += (r.n_local + 63) / 64 * 64;  // keep blocks 1 KB aligned for float4 access
    }
    for (int k = 0; k < h->K; ++k) if (r.emit[k] > h->dep_bound[k]) h->dep_bound[k] = r.emit[k];
    h->rel.push_back(r);
    // the met buffers blended ahead (and the plume mask they were cut to) know nothing of this source
    h->blend_n = 0;
    h->bbox_valid = false;
    return LPM_OK;
}

int32_t lpm_step(lpm_handle *h, int32_t n_steps)
{
    if (!h || n_steps < 0) return fail(h, LPM_ERR_INVALID_ARG, "lpm_step: negative step count");
    if (h->sticky) return h->sticky;
    const bool compact = h->prm.compact != 0;
    StepArgs A;
    base_args(h, A);
    // up to 16 steps per launch; up to 64 when one met buffer serves every step and no sink uses the deposit tables
    const int m_cap = (!compact && h->met.nt == 1 && !A.any_dep) ? kMaxFusedLong : kMaxFused;
    int m_max = h->prm.steps_per_launch > 0 ? h->prm.steps_per_launch : m_cap;
    if (m_max > m_cap) m_max = m_cap;
    if (compact) m_max = 1;
    if (h->met.nt > 1 && m_max > kBlendDepth) m_max = kBlendDepth;  // one time-blended met buffer per fused step
    int64_t left = n_steps;
    while (left > 0) {
        bool fused_bin = false;
        int m = (int)(left < m_max ? left : m_max);
        if (h->prm.bin_every > 0) {
            const uint64_t to_bin = (uint64_t)h->prm.bin_every - h->step % (uint64_t)h->prm.bin_every;
            if ((uint64_t)m > to_bin) m = (int)to_bin;
        }
        A.step0 = h->step;
        for (int s = 0; s < m; ++s) {
            fill_entry(h, h->step + s, A.tab[s]);
            for (int k = 0; k < LPM_MAX_NUCLIDES; ++k) {
                // table units of the deposit increments; R13: Er = growth since the first step of the launch (1 without ground decay)
                StepEntry &e = A.tab[s];
                const double Er = h->prm.ground_decay && k < h->K ? exp(h->lam_dt[k] * s) : 1.0;
                const double sd = (double)A.dep_scale[2 * k] * Er, sw = (double)A.dep_scale[2 * k + 1] * Er;
                e.Gps[k] = (float)((double)e.Gp[k] * sd);
                e.Pd[k] = (float)((double)h->p_dry[k] * sd);
                e.Pw[k] = (float)((double)(float)h->wet_scale[k] * sw);
                e.Oid[k] = (float)(1.0 / sd);
                e.Oiw[k] = (float)(1.0 / sw);
                e.Eg[k] = Er;   // x E0 below, once the launch's first step is final
            }
            // a launch stays inside one met interval: the pair buffer holds snapshots (s, s+1)
            if ((A.tab[s].snap & 0xffff) != (A.tab[0].snap & 0xffff)) { m = s; break; }
        }
        A.m_steps = m;
        if (h->prm.ground_decay) {
            // R13: the map of nuclide k holds activity referred to step dep_ref[k]; an increment of step n enters as
            // inc * exp(lambda (t_n - t_ref)) = inc * E0 * Er(n).  Move the reference before E0 grows large.
            for (int k = 0; k < h->K; ++k) {
                double age = h->lam_dt[k] * (double)(h->step - h->dep_ref[k]);
                if (age > 4.0) {
                    CK(launch_dep_rebase((double *)(h->ws + h->L.dep) + (uint64_t)k * A.dep_stride, A.dep_stride, exp(-age), h->st));
                    h->launches++;
                    h->dep_ref[k] = h->step;
                    age = 0.0;
                }
                const double E0 = exp(age);
                A.dep_inv_scale[2 * k] = E0 / (double)A.dep_scale[2 * k];
                A.dep_inv_scale[2 * k + 1] = E0 / (double)A.dep_scale[2 * k + 1];
                for (int s = 0; s < m; ++s) A.tab[s].Eg[k] *= E0;
            }
        }
        {
            const int rc = ensure_blend(h, A, m, m_max);
            if (rc) return rc;
        }
        A.mask = nullptr;
        if (h->met.nt > 1 && h->step + (uint64_t)m >= h->blend_step0 + (uint64_t)h->blend_n) {
            // the next launch blends again: the step launches below flag the mask tiles that hold their particles
            const int ntx = (h->met.grid.nx + kMaskTile - 1) / kMaskTile, nty = (h->met.grid.ny + kMaskTile - 1) / kMaskTile;
            CK(cudaMemsetAsync(h->ws + h->L.mask, 0, (size_t)ntx * nty, h->st));
            A.mask = (uint8_t *)(h->ws + h->L.mask);
            A.mask_ntx = ntx;
            h->bbox_valid = true;
        } else if (h->met.nt > 1) {
            h->bbox_valid = false;  // (cannot happen before a blend: kept for safety when the coverage logic changes)
        }
        if (compact) {
            InjectArgs I{};
            I.xyzq = A.xyzq; I.q1 = A.q1; I.pid = A.pid; I.ctrl = A.ctrl;
            I.log_slot = (uint64_t *)(h->ws + h->L.injlog) + h->step % kInjLog;
            I.capacity = h->prm.capacity;
            I.K = h->K;
            for (size_t ri = 0; ri < h->rel.size(); ++ri) {
                const Release &r = h->rel[ri];
                const uint64_t b1 = born_local(r, (int64_t)h->step), b0 = born_local(r, (int64_t)h->step - 1);
                if (b1 == b0) continue;
                InjectSpec &sp = I.spec[I.n_spec++];
                sp.rel_index = (int32_t)ri;
                sp.first_pid = r.pid_offset + b0 * r.pid_stride;
                sp.count = b1 - b0;
                sp.pid_stride = r.pid_stride;
                sp.sx = (float)r.src.x; sp.sy = (float)r.src.y; sp.sz = (float)r.src.z;
                for (int k = 0; k < h->K; ++k) sp.q[k] = (float)(r.emit[k] / A.tab[0].G[k]);
            }
            if (sort_enabled(&h->prm)) {
                const uint64_t period = h->prm.gather_sort > 0 ? (uint64_t)h->prm.gather_sort : (uint64_t)h->sort_period;
                if (h->step - h->csort_step >= period) {
                    const int sspan = span_open(h, 2, 0.0);
                    CK(launch_sort_records(A.xyzq, A.q1, A.pid, A.ctrl + 2, h->prm.capacity, A.mg, (uint32_t *)(h->ws + h->L.keys),
                                           (uint32_t *)(h->ws + h->L.hist), (uint32_t *)(h->ws + h->L.partial),
                                           (float4 *)(h->ws + h->L.alt_xyzq), h->K > 1 ? (float *)(h->ws + h->L.alt_q1) : nullptr,
                                           (uint32_t *)(h->ws + h->L.alt_pid), h->st));
                    span_close(h, sspan);
                    h->launches += 6;
                    h->csort_step = h->step;
                }
            }
            CK(launch_inject(I, h->st));
            // unordered store (the records are re-sorted by met cell anyway, B7): hole list + fill instead of the scan
            A.holes = sort_enabled(&h->prm) ? (uint32_t *)(h->ws + h->L.keys) : nullptr;
            const int span = span_open(h, 0, 0.0);
            CK(launch_step(A, h->K, true, h->sms * (h->occ > 0 ? h->occ : 1), h->st));
            if (A.holes) {
                CK(launch_fill_holes(A.xyzq, A.q1, A.pid, A.ctrl, A.holes, (uint32_t *)(h->ws + h->L.alt_pid), (uint32_t *)(h->ws + h->L.alt_xyzq), h->st));
                h->launches += 2;
            }
            span_close(h, span);
            h->launches += 2;
        } else {
            // a8 fused: a launch that ends on a binning step bins its particles itself (lpm_step.cu: bin_tile)
            // (the epilogue is instantiated for the default physics: expected-mass deposition, gridded Kz, uniform levels, no drift)
            fused_bin = h->prm.bin_every > 0 && (h->step + (uint64_t)m) % (uint64_t)h->prm.bin_every == 0 && !A.bern && !A.eq3 && !A.drift &&
                        !h->has_levels;
            A.bin_cnt = nullptr;
            if (fused_bin) {
                const uint64_t cells3 = (uint64_t)h->cg.nx * h->cg.ny * h->cg.nz;
                const int bspan = span_open(h, 1, 0.0);
                CK(cudaMemsetAsync(h->ws + h->L.cnt, 0, (h->L.conc - h->L.cnt) + 8 * cells3 * h->K, h->st));
                span_close(h, bspan);
                A.bin_cnt = (uint32_t *)(h->ws + h->L.cnt);
                A.bin_conc = (double *)(h->ws + h->L.conc);
                A.bin_cells3 = cells3;
                bin_scales(h, h->step + (uint64_t)m, A.bin_scale, A.bin_inv_scale);
            }
            for (const Release &r : h->rel) {
                const uint64_t n = born_local(r, (int64_t)h->step + m - 1);
                if (!n) continue;
                A.base = r.base;
                A.n = n;
                A.n_prev = born_local(r, (int64_t)h->step - 1);
                A.pid_offset = r.pid_offset; A.pid_stride = r.pid_stride;
                A.rel_N = r.N; A.rel_c = r.c ? r.c : 1;
                A.rel_s_start = r.s_start; A.rel_S = r.S;
                for (int k = 0; k < LPM_MAX_NUCLIDES; ++k) A.emit[k] = r.emit[k];
                A.sx = (float)r.src.x; A.sy = (float)r.src.y; A.sz = (float)r.src.z;
                double units = 0.0;
                if (h->timing)
                    for (int s = 0; s < m; ++s) units += (double)born_local(r, (int64_t)h->step + s);
                A.perm = nullptr;
                A.n_perm = 0;
                A.n_live = nullptr;
                A.keys_out = nullptr; A.hist_out = nullptr; A.n_keys = 0;
                if (sort_enabled(&h->prm) && A.n_prev > 0 && (h->prm.gather_sort > 0 || A.n_prev >= kSortAutoMin)) {
                    // the list is kept for `period` model steps (one release: the perm buffer is its own);
                    // particles born since the last sort are walked in slot order behind it
                    uint32_t *perm = perm_half(h, h->perm_cur);
                    uint64_t *live = A.ctrl + kCtrlLive;
                    const bool single = h->rel.size() == 1;
                    const uint64_t period = h->prm.gather_sort > 0 ? (uint64_t)h->prm.gather_sort : (uint64_t)h->sort_period;
                    const uint32_t n_keys = (uint32_t)A.snap_cells + 1u;
                    uint32_t *keys = (uint32_t *)(h->ws + h->L.keys), *hist = (uint32_t *)(h->ws + h->L.hist);
                    if (!single || !h->perm_valid || h->step - h->perm_step >= period || h->perm_n > A.n_prev) {
                        const int sspan = span_open(h, 2, (double)A.n_prev);
                        if (single && h->keys_ready && h->keys_n == A.n_prev && h->keys_step == h->step) {
                            if (h->sort_by_slot) {
                                // keys indexed by slot: the scatter walks the slots in order, each cell's slots end up ascending
                                CK(launch_sort_finish(keys, A.n_prev, n_keys, hist, (uint32_t *)(h->ws + h->L.partial), nullptr, 0, nullptr, perm, live + h->perm_cur, h->st));
                            } else {
                                // the keys stand in the order of the current list (written by the previous launch): build the other one
                                const uint64_t *live_old = live + h->perm_cur;
                                h->perm_cur ^= 1;
                                uint32_t *next = perm_half(h, h->perm_cur);
                                CK(launch_sort_finish(keys, A.n_prev, n_keys, hist, (uint32_t *)(h->ws + h->L.partial), perm, h->perm_n, live_old, next, live + h->perm_cur, h->st));
                                perm = next;
                            }
                            h->launches += 4;
                        } else {
                            CK(launch_sort_by_cell(A.xyzq + r.base, A.n_prev, A.mg, keys, hist, (uint32_t *)(h->ws + h->L.partial), perm, live + h->perm_cur, h->st));
                            h->launches += 5;
                        }
                        span_close(h, sspan);
                        h->perm_n = A.n_prev;
                        h->perm_step = h->step;
                        h->perm_valid = single;
                    }
                    A.perm = perm;
                    A.n_perm = h->perm_n;
                    A.n_live = live + h->perm_cur;
                    // will the next launch sort?  then this one leaves the keys and the histogram
                    h->keys_ready = false;
                    if (single && h->step + (uint64_t)m - h->perm_step >= period) {
                        CK(cudaMemsetAsync(hist, 0, 4ull * n_keys, h->st));
                        A.keys_out = keys; A.hist_out = hist; A.n_keys = n_keys;
                        A.keys_by_slot = h->sort_by_slot ? 1 : 0;
                        h->keys_ready = true;
                        h->keys_n = n;
                        h->keys_step = h->step + (uint64_t)m;
                    }
                }
                CK(cudaMemsetAsync(A.ctrl + 16, 0, 8, h->st));  // tile ticket of the slot kernel
                const int span = span_open(h, fused_bin ? 3 : 0, units);
                CK(launch_step(A, h->K, false, grid_blocks(h, n), h->st));
                span_close(h, span);
                h->launches++;
            }
        }
        h->step += (uint64_t)m;
        left -= m;
        if (h->prm.bin_every > 0 && h->step % (uint64_t)h->prm.bin_every == 0) {
            if (fused_bin) { h->bin_step = h->step; h->binned = true; }
            else { const int rc = do_bin(h); if (rc) return rc; }
            if (h->prm.dose) {
                // P:L108 / Fig. 2b "time integrated dosage": concentration of this binning x the interval it stands for
                const double T = (double)h->prm.bin_every * h->prm.dt, V = h->cg.dx * h->cg.dy * h->cg.dz;
                double sc[LPM_MAX_NUCLIDES] = {0, 0};
                for (int k = 0; k < h->K; ++k) sc[k] = G_of(h, k, h->step) / V * T;
                CK(launch_dose_accum((const double *)(h->ws + h->L.conc), (double *)(h->ws + h->L.dose),
                                     (uint64_t)h->cg.nx * h->cg.ny * h->cg.nz, h->K, sc, h->st));
                h->launches++;
            }
        }
    }
    return LPM_OK;
}

int32_t lpm_bin_now(lpm_handle *h)
{
    if (!h) return LPM_ERR_INVALID_ARG;
    if (h->sticky) return h->sticky;
    return do_bin(h);
}

int32_t lpm_concentration(lpm_handle *h, float *out)
{
    if (!h || !out) return fail(h, LPM_ERR_INVALID_ARG, "lpm_concentration: null");
    if (h->sticky) return h->sticky;
    if (!h->binned || h->bin_step != h->step) { const int rc = do_bin(h); if (rc) return rc; }
    const double V = h->cg.dx * h->cg.dy * h->cg.dz;
    double scale[LPM_MAX_NUCLIDES] = {0, 0};
    for (int k = 0; k < h->K; ++k) scale[k] = G_of(h, k, h->bin_step) / V;
    CK(launch_conc_readout((const double *)(h->ws + h->L.conc), out, (uint64_t)h->cg.nx * h->cg.ny * h->cg.nz, h->K, scale, h->st));
    h->launches++;
    return LPM_OK;
}

int32_t lpm_dose(lpm_handle *h, float *out)
{
    if (!h || !out) return fail(h, LPM_ERR_INVALID_ARG, "lpm_dose: null");
    if (!h->prm.dose) return fail(h, LPM_ERR_STATE, "lpm_dose: params.dose was 0 at lpm_create");
    if (h->sticky) return h->sticky;
    const double one[LPM_MAX_NUCLIDES] = {1.0, 1.0};
    CK(launch_conc_readout((const double *)(h->ws + h->L.dose), out, (uint64_t)h->cg.nx * h->cg.ny * h->cg.nz, h->K, one, h->st));
    h->launches++;
    return LPM_OK;
}

int32_t lpm_counts(lpm_handle *h, uint32_t *out)
{
    if (!h || !out) return fail(h, LPM_ERR_INVALID_ARG, "lpm_counts: null");
    if (h->sticky) return h->sticky;
    if (!h->binned || h->bin_step != h->step) { const int rc = do_bin(h); if (rc) return rc; }
    CK(cudaMemcpyAsync(out, h->ws + h->L.cnt, 4ull * h->cg.nx * h->cg.ny * h->cg.nz, cudaMemcpyDeviceToDevice, h->st));
    return LPM_OK;
}

static int dep_out(lpm_handle *h, float *o32, double *o64)
{
    if (!h || (!o32 && !o64)) return fail(h, LPM_ERR_INVALID_ARG, "lpm_deposition: null");
    if (h->sticky) return h->sticky;
    double scale[LPM_MAX_NUCLIDES] = {0, 0};
    for (int k = 0; k < h->K; ++k)   // per cell area; R13: the ground decay since the map's reference time
        scale[k] = (h->prm.ground_decay ? exp(-h->lam_dt[k] * (double)(h->step - h->dep_ref[k])) : 1.0) / (h->cg.dx * h->cg.dy);
    CK(launch_dep_readout((const double *)(h->ws + h->L.dep), o32, o64, (uint64_t)h->cg.nx * h->cg.ny, h->K, scale, h->st));
    h->launches++;
    return LPM_OK;
}

int32_t lpm_deposition(lpm_handle *h, float *out) { return dep_out(h, out, nullptr); }
int32_t lpm_deposition_f64(lpm_handle *h, double *out) { return dep_out(h, nullptr, out); }

int32_t lpm_step_index(lpm_handle *h, uint64_t *s)
{
    if (!h || !s) return LPM_ERR_INVALID_ARG;
    *s = h->step;
    return LPM_OK;
}

int32_t lpm_mass_scale(lpm_handle *h, double *scale)
{
    if (!h || !scale) return LPM_ERR_INVALID_ARG;
    for (int k = 0; k < h->K; ++k) scale[k] = G_of(h, k, h->step);
    return LPM_OK;
}

static uint64_t slots_in_use(const lpm_handle *h)
{
    uint64_t n = 0;
    for (const Release &r : h->rel) {
        const uint64_t b = born_local(r, (int64_t)h->step - 1);
        if (b && r.base + b > n) n = r.base + b;
    }
    return n;
}

int32_t lpm_num_active(lpm_handle *h, uint64_t *n)
{
    if (!h || !n) return LPM_ERR_INVALID_ARG;
    if (h->sticky) return h->sticky;
    if (h->prm.compact) {
        CK(cudaMemcpyAsync(n, (uint64_t *)(h->ws + h->L.ctrl) + 2, 8, cudaMemcpyDeviceToHost, h->st));
        CK(cudaStreamSynchronize(h->st));
    } else {
        *n = slots_in_use(h);
    }
    return LPM_OK;
}

int32_t lpm_get_particles(lpm_handle *h, void *xyzq, float *q1, uint32_t *pid, uint8_t *status, uint64_t *n_host)
{
    if (!h || !n_host) return fail(h, LPM_ERR_INVALID_ARG, "lpm_get_particles: null");
    if (h->sticky) return h->sticky;
    uint64_t n = 0;
    const int rc = lpm_num_active(h, &n);
    if (rc) return rc;
    *n_host = n;
    if (!n) return LPM_OK;
    if (xyzq || status) {
        CK(launch_export((const float4 *)(h->ws + h->L.xyzq), h->K > 1 ? (const float *)(h->ws + h->L.q1) : nullptr, n, nullptr, (float4 *)xyzq, status, h->st));
        h->launches++;
    }
    if (q1 && h->K > 1) CK(cudaMemcpyAsync(q1, h->ws + h->L.q1, 4 * n, cudaMemcpyDeviceToDevice, h->st));
    if (pid) {
        if (h->prm.compact) CK(cudaMemcpyAsync(pid, h->ws + h->L.pid, 4 * n, cudaMemcpyDeviceToDevice, h->st));
        else {
            // slot-addressed mode: ids are implied by the slot: pid_offset + l * pid_stride inside each release block
            // (the padding slots between two blocks report 0)
            CK(cudaMemsetAsync(pid, 0, 4 * n, h->st));
            for (const Release &r : h->rel) {
                const uint64_t b = born_local(r, (int64_t)h->step - 1);
                if (!b) continue;
                CK(launch_iota(pid + r.base, b, r.pid_offset, r.pid_stride, h->st));
                h->launches++;
            }
        }
    }
    return LPM_OK;
}

int32_t lpm_set_particles(lpm_handle *h, const void *xyzq, const float *q1, const uint32_t *pid, const uint8_t *status,
                          uint64_t n, uint64_t step_index)
{
    if (!h || !xyzq || (h->K > 1 && !q1)) return fail(h, LPM_ERR_INVALID_ARG, "lpm_set_particles: null");
    if (n > h->prm.capacity) return fail(h, LPM_ERR_CAPACITY, "lpm_set_particles: n exceeds capacity");
    if (h->sticky) return h->sticky;
    uint64_t id_off = 0, id_stride = 1;
    if (!h->prm.compact && pid && n) {
        // slot-addressed store: ids are implied by the slot, so the given ids must be offset + l * stride (what
        // lpm_get_particles reports for one release); offset and stride are read back from the first two entries
        uint32_t two[2] = {0, 0};
        CK(cudaMemcpyAsync(two, pid, n > 1 ? 8 : 4, cudaMemcpyDeviceToHost, h->st));
        CK(cudaStreamSynchronize(h->st));
        id_off = two[0];
        if (n > 1) {
            if (two[1] <= two[0]) return fail(h, LPM_ERR_INVALID_ARG, "lpm_set_particles: slot-addressed store needs ascending affine ids");
            id_stride = two[1] - two[0];
        }
        if (id_off + (n - 1) * id_stride >= (1ull << 32)) return fail(h, LPM_ERR_INVALID_ARG, "lpm_set_particles: particle ids must stay below 2^32");
        uint32_t *bad = (uint32_t *)(h->ws + h->L.air);
        uint32_t bad_h = 0;
        CK(cudaMemsetAsync(bad, 0, 4, h->st));
        CK(launch_check_affine(pid, n, id_off, id_stride, bad, h->st));
        h->launches++;
        CK(cudaMemcpyAsync(&bad_h, bad, 4, cudaMemcpyDeviceToHost, h->st));
        CK(cudaStreamSynchronize(h->st));
        if (bad_h) return fail(h, LPM_ERR_INVALID_ARG, "lpm_set_particles: ids are implied by the slot unless compact=1: pid must be offset + l*stride");
    }
    if (n) {
        CK(cudaMemcpyAsync(h->ws + h->L.xyzq, xyzq, 16 * n, cudaMemcpyDeviceToDevice, h->st));
        if (h->K > 1) CK(cudaMemcpyAsync(h->ws + h->L.q1, q1, 4 * n, cudaMemcpyDeviceToDevice, h->st));
        if (status) { CK(launch_import((float4 *)(h->ws + h->L.xyzq), n, status, h->st)); h->launches++; }
    }
    if (h->prm.compact) {
        if (n) {
            if (pid) CK(cudaMemcpyAsync(h->ws + h->L.pid, pid, 4 * n, cudaMemcpyDeviceToDevice, h->st));
            else { CK(launch_iota((uint32_t *)(h->ws + h->L.pid), n, 0, 1, h->st)); h->launches++; }
        }
        // the look-back tile states carry the step index as their epoch: a clock moved backwards must not meet old ones
        CK(cudaMemsetAsync(h->ws + h->L.tile, 0, 8 * (h->prm.capacity / kScanTile + 2), h->st));
        uint64_t ctrl[3] = {n, 0, n};
        CK(cudaMemcpyAsync(h->ws + h->L.ctrl, ctrl, sizeof(ctrl), cudaMemcpyHostToDevice, h->st));
        CK(cudaStreamSynchronize(h->st));
    } else {
        h->rel.clear();
        Release r{};
        r.fixed = true; r.n_local = n; r.pid_offset = id_off; r.pid_stride = id_stride; r.S = 1;
        h->rel.push_back(r);
        h->next_base = n;
    }
    if (h->prm.ground_decay) {
        // R13: the clock may jump (restart from a checkpoint): bring each map to the present first, then regard it as
        // the ground activity at the new step index
        for (int k = 0; k < h->K; ++k) {
            const double age = h->lam_dt[k] * (double)(h->step - h->dep_ref[k]);
            if (age > 0.0) {
                const uint64_t c2 = (uint64_t)h->cg.nx * h->cg.ny;
                CK(launch_dep_rebase((double *)(h->ws + h->L.dep) + (uint64_t)k * c2, c2, exp(-age), h->st));
                h->launches++;
            }
            h->dep_ref[k] = step_index;
        }
    }
    h->step = step_index;
    h->binned = false;
    h->perm_valid = false;
    h->keys_ready = false;
    h->bbox_valid = false;
    h->blend_n = 0;
    h->csort_step = step_index;
    if (n) {  // the installed activities bound the deposit increments from now on
        float *mx = (float *)(h->ws + h->L.air);
        float mq[2] = {0.f, 0.f};
        CK(cudaMemsetAsync(mx, 0, 8, h->st));
        CK(launch_qmax((const float4 *)(h->ws + h->L.xyzq), h->K > 1 ? (const float *)(h->ws + h->L.q1) : nullptr, n, h->K, mx, h->st));
        h->launches++;
        CK(cudaMemcpyAsync(mq, mx, 8, cudaMemcpyDeviceToHost, h->st));
        CK(cudaStreamSynchronize(h->st));
        for (int k = 0; k < h->K; ++k) {
            const double b = (double)mq[k] * G_of(h, k, step_index);
            if (!h->prm.compact || b > h->dep_bound[k]) h->dep_bound[k] = b;
        }
    }
    return LPM_OK;
}

int32_t lpm_ledger(lpm_handle *h, double *out)
{
    if (!h || !out) return fail(h, LPM_ERR_INVALID_ARG, "lpm_ledger: null");
    if (h->sticky) return h->sticky;
    double *air = (double *)(h->ws + h->L.air);
    CK(cudaMemsetAsync(air, 0, 16, h->st));
    if (h->prm.compact) {
        CK(launch_airborne((const float4 *)(h->ws + h->L.xyzq), h->K > 1 ? (const float *)(h->ws + h->L.q1) : nullptr, 0,
                           (const uint64_t *)(h->ws + h->L.ctrl) + 2, h->K, air, h->st));
        h->launches++;
    } else {
        for (const Release &r : h->rel) {
            const uint64_t n = born_local(r, (int64_t)h->step - 1);
            if (!n) continue;
            CK(launch_airborne((const float4 *)(h->ws + h->L.xyzq) + r.base,
                               h->K > 1 ? (const float *)(h->ws + h->L.q1) + r.base : nullptr, n, nullptr, h->K, air, h->st));
            h->launches++;
        }
    }
    double led[LPM_MAX_NUCLIDES * 8], a2[2];
    uint64_t ctrl[32];
    CK(cudaMemcpyAsync(led, h->ws + h->L.ledger, sizeof(led), cudaMemcpyDeviceToHost, h->st));
    CK(cudaMemcpyAsync(a2, air, 16, cudaMemcpyDeviceToHost, h->st));
    CK(cudaMemcpyAsync(ctrl, h->ws + h->L.ctrl, sizeof(ctrl), cudaMemcpyDeviceToHost, h->st));
    CK(cudaStreamSynchronize(h->st));
    for (int k = 0; k < h->K; ++k) {
        double emitted = 0.0;
        for (size_t ri = 0; ri < h->rel.size(); ++ri) {
            const Release &r = h->rel[ri];
            if (r.fixed) continue;
            const uint64_t born = h->prm.compact ? ctrl[8 + ri] : born_local(r, (int64_t)h->step - 1);
            emitted += r.emit[k] * (double)born;
        }
        double *o = out + k * LPM_LEDGER_FIELDS;
        o[0] = emitted;
        o[1] = a2[k] * G_of(h, k, h->step);
        o[2] = led[k * 8 + 2]; o[3] = led[k * 8 + 3]; o[4] = led[k * 8 + 4]; o[5] = led[k * 8 + 5]; o[6] = led[k * 8 + 6];
    }
    return LPM_OK;
}

int32_t lpm_injected(lpm_handle *h, uint64_t step, uint64_t *n)
{
    if (!h || !n) return LPM_ERR_INVALID_ARG;
    if (h->sticky) return h->sticky;
    *n = 0;
    if (step >= h->step) return LPM_OK;
    if (h->prm.compact) {
        if (h->step - step > kInjLog) return fail(h, LPM_ERR_INVALID_ARG, "lpm_injected: step fell out of the log ring");
        CK(cudaMemcpyAsync(n, (uint64_t *)(h->ws + h->L.injlog) + step % kInjLog, 8, cudaMemcpyDeviceToHost, h->st));
        CK(cudaStreamSynchronize(h->st));
    } else {
        for (const Release &r : h->rel) *n += born_local(r, (int64_t)step) - born_local(r, (int64_t)step - 1);
    }
    return LPM_OK;
}

int32_t lpm_upload_meteo(lpm_handle *h, int32_t first, int32_t n_snap, const void *src)
{
    if (!h || !src || first < 0 || n_snap < 1 || first + n_snap > h->met.nt) return fail(h, LPM_ERR_INVALID_ARG, "lpm_upload_meteo: null or range");
    if (h->sticky) return h->sticky;
    const lpm_grid &g = h->met.grid;
    const uint64_t snap_bytes = 16ull * g.nx * g.ny * g.nz;
    CK(cudaMemcpyAsync((char *)h->met.fields_dev + (uint64_t)first * snap_bytes, src, snap_bytes * (uint64_t)n_snap,
                       cudaMemcpyHostToDevice, h->st));
    if (h->pair_snap >= first - 1 && h->pair_snap < first + n_snap) h->pair_snap = -1;  // the pair buffer is stale
    h->blend_n = 0;                                                                    // and so are the blended fields
    return LPM_OK;
}

int32_t lpm_concentration_host(lpm_handle *h, float *out)
{
    if (!h || !out) return fail(h, LPM_ERR_INVALID_ARG, "lpm_concentration_host: null");
    float *stage = (float *)(h->ws + h->L.stage);
    const int rc = lpm_concentration(h, stage);
    if (rc) return rc;
    CK(cudaMemcpyAsync(out, stage, 4ull * h->cg.nx * h->cg.ny * h->cg.nz * h->K, cudaMemcpyDeviceToHost, h->st));
    CK(cudaStreamSynchronize(h->st));
    return LPM_OK;
}

int32_t lpm_deposition_host(lpm_handle *h, float *out)
{
    if (!h || !out) return fail(h, LPM_ERR_INVALID_ARG, "lpm_deposition_host: null");
    float *stage = (float *)(h->ws + h->L.stage);
    const int rc = lpm_deposition(h, stage);
    if (rc) return rc;
    CK(cudaMemcpyAsync(out, stage, 4ull * h->cg.nx * h->cg.ny * h->K, cudaMemcpyDeviceToHost, h->st));
    CK(cudaStreamSynchronize(h->st));
    return LPM_OK;
}

int32_t lpm_set_timing(lpm_handle *h, int32_t enable)
{
    if (!h) return LPM_ERR_INVALID_ARG;
    CK(cudaStreamSynchronize(h->st));
    spans_collect(h);
    h->timing = enable != 0;
    for (int i = 0; i < 5; ++i) { h->t_ms[i] = 0.0; h->t_units[i] = 0.0; h->t_launches[i] = 0; }
    CK(cudaMemcpyAsync(&h->t_base, (uint64_t *)(h->ws + h->L.ctrl) + kCtrlSteps, 8, cudaMemcpyDeviceToHost, h->st));
    CK(cudaMemcpyAsync(&h->t_base_bin, (uint64_t *)(h->ws + h->L.ctrl) + kCtrlBinned, 8, cudaMemcpyDeviceToHost, h->st));
    CK(cudaStreamSynchronize(h->st));
    return LPM_OK;
}

int32_t lpm_get_timing(lpm_handle *h, double *out)
{
    if (!h || !out) return LPM_ERR_INVALID_ARG;
    CK(cudaStreamSynchronize(h->st));
    spans_collect(h);
    out[0] = h->t_ms[0]; out[1] = (double)h->t_launches[0];
    out[2] = h->t_ms[1]; out[3] = (double)h->t_launches[1];
    out[4] = h->t_units[0]; out[5] = h->t_units[1];
    out[6] = h->t_ms[2]; out[7] = (double)h->t_launches[2];
    out[9] = h->t_ms[3]; out[10] = (double)h->t_launches[3]; out[11] = h->t_ms[4];
    out[12] = h->t_units[3]; out[13] = h->t_units[4];
    out[8] = h->t_units[0];   // born particles x steps (host count, R9): includes particles that have left the domain
    // what the kernels counted themselves: particle-steps executed (born AND active), particles binned (active, in the grid)
    uint64_t now[2] = {0, 0};
    CK(cudaMemcpyAsync(&now[0], (uint64_t *)(h->ws + h->L.ctrl) + kCtrlSteps, 8, cudaMemcpyDeviceToHost, h->st));
    CK(cudaMemcpyAsync(&now[1], (uint64_t *)(h->ws + h->L.ctrl) + kCtrlBinned, 8, cudaMemcpyDeviceToHost, h->st));
    CK(cudaStreamSynchronize(h->st));
    out[4] = (double)(now[0] - h->t_base);
    out[5] = (double)(now[1] - h->t_base_bin);
    return LPM_OK;
}

int32_t lpm_touched_cells(lpm_handle *h, uint64_t *n)
{
    if (!h || !n) return LPM_ERR_INVALID_ARG;
    if (h->sticky) return h->sticky;
    if (!h->binned) return fail(h, LPM_ERR_STATE, "lpm_touched_cells: nothing has been binned yet");
    uint64_t *dst = (uint64_t *)(h->ws + h->L.ctrl) + kCtrlTouched;
    CK(cudaMemsetAsync(dst, 0, 8, h->st));
    CK(launch_count_nonzero((const uint32_t *)(h->ws + h->L.cnt), (uint64_t)h->cg.nx * h->cg.ny * h->cg.nz, dst, h->st));
    h->launches++;
    CK(cudaMemcpyAsync(n, dst, 8, cudaMemcpyDeviceToHost, h->st));
    CK(cudaStreamSynchronize(h->st));
    return LPM_OK;
}

int32_t lpm_texel_pairs(lpm_handle *h, int32_t *on)
{
    if (!h || !on) return LPM_ERR_INVALID_ARG;
    *on = h->zpair ? 1 : 0;
    return LPM_OK;
}

int32_t lpm_launch_count(lpm_handle *h, uint64_t *n)
{
    if (!h || !n) return LPM_ERR_INVALID_ARG;
    *n = h->launches;
    return LPM_OK;
}

static int dev_ok()
{
    int ndev = 0;
    return cudaGetDeviceCount(&ndev) == cudaSuccess && ndev > 0;
}

int32_t lpm_probe(int32_t kind, uint64_t footprint, void *scratch, uint64_t scratch_bytes, int32_t reps, double *ops, void *st)
{
    if (!scratch || !ops || kind < 0 || kind > LPM_PROBE_GATHER32 || scratch_bytes < (1u << 20) || reps < 1 || ((uintptr_t)scratch & 15))
        return LPM_ERR_INVALID_ARG;
    if (!dev_ok()) return LPM_ERR_NO_DEVICE;
    if (footprint == 0 || footprint > scratch_bytes) footprint = scratch_bytes;
    if ((kind == LPM_PROBE_GATHER || kind == LPM_PROBE_GATHER32) && footprint > scratch_bytes - 64) footprint = scratch_bytes - 64;
    return run_probe(kind, footprint, scratch, scratch_bytes, reps, ops, (cudaStream_t)st) == cudaSuccess ? LPM_OK : LPM_ERR_CUDA;
}

int32_t lpm_test_philox(uint64_t seed, uint64_t step, uint32_t stream, uint64_t pid0, uint64_t n, uint32_t *out, void *st)
{
    if (!out) return LPM_ERR_INVALID_ARG;
    if (!dev_ok()) return LPM_ERR_NO_DEVICE;
    return launch_test_philox(seed, step, stream, pid0, n, out, (cudaStream_t)st) == cudaSuccess ? LPM_OK : LPM_ERR_CUDA;
}

int32_t lpm_test_normals(uint64_t seed, uint64_t step, uint64_t pid0, uint64_t n, float *out, void *st)
{
    if (!out) return LPM_ERR_INVALID_ARG;
    if (!dev_ok()) return LPM_ERR_NO_DEVICE;
    return launch_test_normals(seed, step, pid0, n, out, (cudaStream_t)st) == cudaSuccess ? LPM_OK : LPM_ERR_CUDA;
}

int32_t lpm_test_curand_philox(uint64_t seed, uint64_t step, uint64_t pid0, uint64_t n, uint32_t *out, void *st)
{
    if (!out) return LPM_ERR_INVALID_ARG;
    if (!dev_ok()) return LPM_ERR_NO_DEVICE;
    return launch_test_curand_philox(seed, step, pid0, n, out, (cudaStream_t)st) == cudaSuccess ? LPM_OK : LPM_ERR_CUDA;
}

int32_t lpm_test_box_muller(const uint32_t *r, uint64_t n, float *out, void *st)
{
    if (!r || !out || ((uintptr_t)r & 15)) return LPM_ERR_INVALID_ARG;
    if (!dev_ok()) return LPM_ERR_NO_DEVICE;
    return launch_test_box_muller(r, n, out, (cudaStream_t)st) == cudaSuccess ? LPM_OK : LPM_ERR_CUDA;
}

int32_t lpm_test_sample(const lpm_meteo *met, double t, const void *xyz, uint64_t n, void *out, void *st)
{
    if (!met || !grid_ok(&met->grid) || !met->fields_dev || !xyz || !out || met->nt < 1) return LPM_ERR_INVALID_ARG;
    if (!dev_ok()) return LPM_ERR_NO_DEVICE;
    lpm_handle tmp{};
    tmp.met = *met;
    tmp.prm.dt = 1.0;
    tmp.K = 0;
    StepEntry e;
    // fill_entry evaluates the time weight at t = n * dt; use dt = t, n = 1
    tmp.prm.dt = t;
    fill_entry(&tmp, 1, e);
    const lpm_grid &g = met->grid;
    const uint64_t cells = (uint64_t)g.nx * g.ny * g.nz;
    const float4 *f = (const float4 *)met->fields_dev;
    cudaStream_t s = (cudaStream_t)st;
    const int sn = e.snap & 0xffff;
    // the same path as lpm_step: z-fastest (pair ->) blended buffer, then the step kernel's sampling
    void *pair = nullptr;
    float4 *blend = nullptr;
    if (cudaMalloc((void **)&blend, 16 * cells + 16) != cudaSuccess) return LPM_ERR_CUDA;
    cudaMemsetAsync(blend + cells, 0, 16, s);  // pad texel (read with weight 0 when nz = 1)
    cudaError_t rc;
    if (met->nt > 1) {
        if (cudaMalloc(&pair, 32 * cells) != cudaSuccess) { cudaFree(blend); return LPM_ERR_CUDA; }
        BlendBox box{};
        box.nx = g.nx; box.ny = g.ny; box.nz = g.nz;
        rc = launch_pair_repack(f + (uint64_t)sn * cells, f + (uint64_t)(sn + 1) * cells, pair, g.nx, g.ny, g.nz, nullptr, s);
        if (rc == cudaSuccess) rc = launch_blend(pair, blend, cells, 1, &e.a, &box, false, s);
    } else {
        rc = launch_transpose(f, blend, g.nx, g.ny, g.nz, s);
    }
    float lev[kMaxLevels];
    if (met->z_levels_host) {
        if (g.nz > kMaxLevels) { cudaFree(blend); if (pair) cudaFree(pair); return LPM_ERR_INVALID_ARG; }
        for (int k = 0; k < g.nz; ++k) lev[k] = (float)met->z_levels_host[k];
    }
    if (rc == cudaSuccess) rc = launch_test_sample(blend, gridf(g, true, met->z_levels_host ? lev : nullptr), (float)met->kz_min, (const float4 *)xyz, n, (float4 *)out, s);
    const cudaError_t rs = cudaStreamSynchronize(s);
    if (rc == cudaSuccess) rc = rs;
    cudaFree(blend);
    if (pair) cudaFree(pair);
    return rc == cudaSuccess ? LPM_OK : LPM_ERR_CUDA;
}

}  // extern "C"

// ------------------------------------------------------------------ lpm_sample_static: met sampling without an allocation
//
// For callers that cannot call cudaMalloc (all device memory owned by a host application's pool, or a loop that cannot
// afford the device-wide synchronisation of cudaMalloc / cudaFree): the two temporaries of the sampling path live in the
// library image.  One array per loaded module = per GPU, shared by every call, never freed.
//   [0, 16 * (cells + 1))                       time-blended z-fastest field + the zero pad texel behind it
//   [kStaticPairAt, kStaticPairAt + 32 * cells)  interleaved snapshot pair of the met interval (nt > 1 only)
// g_sample_scratch is a HOST-SIDE STAND-IN for the device array: host code must never hand its name (or &name) to a
// kernel as a pointer.  The device address comes from cudaGetSymbolAddress, once per device, below.
static_assert(LPM_SAMPLE_STATIC_MAX_CELLS % 16 == 0, "the pair buffer starts 256-byte aligned");
constexpr uint64_t kStaticPairAt = 16ull * LPM_SAMPLE_STATIC_MAX_CELLS + 256ull;
static_assert(kStaticPairAt + 32ull * LPM_SAMPLE_STATIC_MAX_CELLS == LPM_SAMPLE_STATIC_BYTES, "lpm.h states the size of the array");
static __device__ __align__(256) unsigned char g_sample_scratch[LPM_SAMPLE_STATIC_BYTES];

namespace {

constexpr int kStaticMaxDevices = 64;
std::mutex g_static_mu;
unsigned char *g_static_addr[kStaticMaxDevices] = {};   // device address of g_sample_scratch on device d; null = not looked up yet

// Device address of the scratch array on the CURRENT device.  First call per device: cudaGetSymbolAddress (this is the
// set-up step lpm.h tells the caller to get out of the way early); afterwards a table look-up.
cudaError_t static_scratch(unsigned char **p)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kStaticMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (!g_static_addr[dev]) {
        void *q = nullptr;
        e = cudaGetSymbolAddress(&q, g_sample_scratch);
        if (e != cudaSuccess) return e;
        if (!q || ((uintptr_t)q & 255)) return cudaErrorInvalidSymbol;
        g_static_addr[dev] = (unsigned char *)q;
    }
    *p = g_static_addr[dev];
    return cudaSuccess;
}

}  // namespace

extern "C" int32_t lpm_sample_static(const lpm_meteo *met, double t, const void *xyz, uint64_t n, void *out, void *st)
{
    if (!met || !grid_ok(&met->grid) || !met->fields_dev || !xyz || !out || met->nt < 1) return LPM_ERR_INVALID_ARG;
    const lpm_grid &g = met->grid;
    if (met->z_levels_host && g.nz > kMaxLevels) return LPM_ERR_INVALID_ARG;
    const uint64_t cells = (uint64_t)g.nx * g.ny * g.nz;
    if (cells > LPM_SAMPLE_STATIC_MAX_CELLS) return LPM_ERR_WORKSPACE_TOO_SMALL;   // the built-in array is this call's workspace
    if (!dev_ok()) return LPM_ERR_NO_DEVICE;
    unsigned char *scratch = nullptr;
    if (static_scratch(&scratch) != cudaSuccess) return LPM_ERR_CUDA;
    float4 *blend = (float4 *)scratch;
    void *pair = scratch + kStaticPairAt;

    lpm_handle tmp{};
    tmp.met = *met;
    tmp.K = 0;
    tmp.prm.dt = t;   // fill_entry evaluates the time weight at n * dt: dt = t, n = 1
    StepEntry e;
    fill_entry(&tmp, 1, e);
    const float4 *f = (const float4 *)met->fields_dev;
    cudaStream_t s = (cudaStream_t)st;
    const int sn = e.snap & 0xffff;
    // The array still holds the last call's field (perhaps of a bigger grid).  Everything below [0, 16 * cells) and the
    // pair buffer is overwritten before it is read; the pad texel at `cells` is read with weight 0 when nz = 1 and must
    // not hold a NaN / Inf left behind by an earlier, larger field: cleared on every call.
    cudaError_t rc = cudaMemsetAsync(blend + cells, 0, 16, s);
    if (rc == cudaSuccess) {
        if (met->nt > 1) {
            BlendBox box{};
            box.nx = g.nx; box.ny = g.ny; box.nz = g.nz;
            rc = launch_pair_repack(f + (uint64_t)sn * cells, f + (uint64_t)(sn + 1) * cells, pair, g.nx, g.ny, g.nz, nullptr, s);
            if (rc == cudaSuccess) rc = launch_blend(pair, blend, cells, 1, &e.a, &box, false, s);
        } else {
            rc = launch_transpose(f, blend, g.nx, g.ny, g.nz, s);
        }
    }
    float lev[kMaxLevels];
    if (met->z_levels_host)
        for (int k = 0; k < g.nz; ++k) lev[k] = (float)met->z_levels_host[k];
    if (rc == cudaSuccess)
        rc = launch_test_sample(blend, gridf(g, true, met->z_levels_host ? lev : nullptr), (float)met->kz_min, (const float4 *)xyz, n,
                                (float4 *)out, s);
    return rc == cudaSuccess ? LPM_OK : LPM_ERR_CUDA;
}
