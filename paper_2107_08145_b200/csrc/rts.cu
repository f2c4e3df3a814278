// rts.cu -- host side of the C-ABI in include/rts.h: ray geometry, sweep units, planner,
// workspace layout, launches.  All arithmetic of the path runs in the kernels of
// rts_kernels.cuh / rts_sweep.cuh; nothing here (or anywhere in the product) touches oracle/.
#include "../../include/rts.h"
#include "rts_kernels.cuh"
// the sweep kernel twice (see the end of rts_sweep.cuh): fixed pass count, and one pass per launch with error words
#define RTS_TOLM 0
#define RTS_MODE_NS fixedp
#include "rts_sweep.cuh"
#undef RTS_TOLM
#undef RTS_MODE_NS
#define RTS_TOLM 1
#define RTS_MODE_NS tolp
#include "rts_sweep.cuh"
#undef RTS_TOLM
#undef RTS_MODE_NS
#include "rts_scatter.cuh"

// Scratch of the entry point that allocates nothing (rts_scatter_solve_static): a file-scope device array, held by
// every GPU that loads this library until the process exits.  In host code the name below is a host-side stand-in,
// NOT a device address: host code takes the address once per device with cudaGetSymbolAddress (resolve_static_scratch,
// called at set-up by rts_create with that device current) and hands that pointer to the kernel.
#define RTS_SCATTER_STATIC_BYTES_IMPL (16u << 20)
static __device__ __align__(256) unsigned char g_scatter_scratch[RTS_SCATTER_STATIC_BYTES_IMPL];

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <cstdlib>
#include <mutex>
#include <string>
#include <vector>

using namespace rts;

namespace {

struct HostRay {
    double mu[3];
    double w;
    int march, dir, su, sv, slot, up, itop;
    double ds, fu, fv;
};

struct TypePlan {        // per march axis
    int n_m = 0, n_u = 0, n_v = 0;
    int WU = 0, WV = 0, ntu = 0, ntv = 0;
    int userWU = 0, userWV = 0;
    int ng = 2;          // ray groups (same su) per unit: 2, or 1 where a plane with all four rays does not fit
    int nstage = 3;      // depth of the coefficient ring
    int rc = 4;          // rows per strip
    int items = 0;       // strips of one ray of a full tile (halo included)
};

struct HostUnit {
    UnitDesc d;
    size_t off_xex, off_g, off_part, off_lp;   // workspace offsets of its exchange planes, seam histories, partial heating, last planes
};

}  // namespace

struct rts_ctx {
    int nx = 0, ny = 0, nz = 0, nb = 0, nbp = 0;   // nbp = band pairs
    double h[3] = {0, 0, 0};
    int npass = 3;
    bool thick_skip = true;
    unsigned solve_seq = 0;            // sweep launches on this context (tags of the exchange words)
    // error-controlled iteration (NEXT #3): one pass per launch until the seam faces change by <= tol * max|I|
    int tol_max_passes = 0;            // 0: off (fixed number of passes in one launch)
    double tol = 0.0;
    bool warm = false;                 // keep the seam state between solves
    int nplain = 0;                    // partial-heating buffers in the x-fastest layout (summed first by the finalize kernel)
    int device = 0;                    // the device this context was created on
    void* static_scratch = nullptr;    // device address of g_scatter_scratch on that device (null: static_scratch_err says why)
    cudaError_t static_scratch_err = cudaSuccess;
    std::vector<ScatRay> scat_rays;    // ray constants of the last rts_scatter_solve (kept until its copy has run)
    int pass_counter = 0;              // passes the seam state has seen (0: cold)
    int passes_used = 0;
    float relerr_last = 0.f;
    size_t off_errw = 0;
    int shard_rank = 0, shard_n = 1;   // this context sweeps the units u with u % shard_n == shard_rank (rts_set_shard)
    int units_all = 0;                 // sweep units of the whole problem
    bool flux = false;           // radiative flux wanted (rts_enable_flux): three more partial fields per unit
    double tau0 = 0.1;           // blend scale of the flux-divergence heating
    std::vector<HostRay> rays;
    int n_up = 0;
    // tables
    bool have_tables = false;
    int nT = 0, nP = 0;
    double logT_min = 0, logT_max = 0, logP_min = 0, logP_max = 0;
    float* d_logkappa = nullptr;
    float* d_bandfrac = nullptr;
    // device facts
    int sm_count = 0, max_smem_optin = 0;
    int user_ctas_per_sm = 0, user_K = 0, user_threads = 0, user_nstage = 0, user_ng = 0, user_rc = 0;
    SweepMaps maps;
    void* encode_fn = nullptr;    // cuTensorMapEncodeTiled
    // plan
    bool planned = false;
    TypePlan tp[3];
    std::vector<HostUnit> units;
    int total_tickets = 0, grid = 0, K = KMAX, pitch = 56;
    int ctas_per_sm = 0, threads = 256, smem_bytes = 0;
    int PX = 0, PY = 0, PYR = 0;
    size_t ws_bytes = 0;
    // workspace offsets
    size_t off_coefA = 0, off_coefB = 0, off_partptr = 0, off_ksum = 0, off_kmin = 0, off_lev = 0, off_kstar = 0, off_mthick = 0, off_mthick_b = 0, off_abort = 0,
           off_units = 0, off_bar = 0, off_stage_in = 0, off_stage_out = 0;
    int nblk_a = 0;
    // workspace
    unsigned char* ws = nullptr;
    size_t ws_have = 0;
    bool maps_ready = false;
    cudaEvent_t ev = nullptr;
    bool timing = false;
    cudaEvent_t tev[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};
    cudaStream_t copy_stream = nullptr;        // rts_solve_host: copies overlap the kernels
    cudaEvent_t hev[10] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    std::string err;
};

namespace {

std::string g_create_err = "null context";   // failures of rts_create (no ctx to hold the text)

int fail(rts_ctx* c, int code, const std::string& msg)
{
    if (c) c->err = msg; else g_create_err = msg;
    return code;
}
#define CUDA_TRY(c, expr)                                                                         \
    do {                                                                                          \
        cudaError_t e_ = (expr);                                                                  \
        if (e_ != cudaSuccess)                                                                    \
            return fail((c), RTS_ECUDA, std::string(#expr) + ": " + cudaGetErrorString(e_));      \
    } while (0)

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// Ray geometry (reading R3): the characteristic leaves the upwind cell through the
// face reached first; ties prefer z, then y, then x.
int ray_geometry(const double h[3], HostRay& r)
{
    double t[3];
    for (int a = 0; a < 3; ++a) t[a] = (r.mu[a] != 0.0) ? h[a] / std::fabs(r.mu[a]) : HUGE_VAL;
    if (r.mu[2] == 0.0) return -1;
    int as = 2;
    if (t[1] < t[as]) as = 1;
    if (t[0] < t[as]) as = 0;
    r.march = as;
    r.ds = t[as];
    r.dir = (r.mu[as] >= 0.0) ? 1 : -1;
    const int ua = (as == 0) ? 1 : 0;          // unit-stride transverse axis
    const int va = (as == 2) ? 1 : 2;          // other transverse axis
    r.su = (r.mu[ua] >= 0.0) ? 1 : -1;
    r.sv = (r.mu[va] >= 0.0) ? 1 : -1;
    r.fu = r.ds * std::fabs(r.mu[ua]) / h[ua];
    r.fv = r.ds * std::fabs(r.mu[va]) / h[va];
    r.slot = ((r.su < 0) ? 1 : 0) + ((r.sv < 0) ? 2 : 0);
    r.up = (r.mu[2] > 0.0) ? 1 : 0;
    return 0;
}

// Bilinear weights as fp32 numbers that sum to 1 EXACTLY: the three smaller ones are rounded
// to multiples of 2^-24, the largest is 1 minus their sum.  A partition of unity that is only
// accurate to an ulp biases the carried intensity by ~6e-8 per step, which accumulates over
// hundreds of steps ("precision").
void make_ray_consts(const HostRay& r, RayC& rc)
{
    double w[4] = {(1 - r.fu) * (1 - r.fv), r.fu * (1 - r.fv), (1 - r.fu) * r.fv, r.fu * r.fv};
    int big = 0;
    for (int q = 1; q < 4; ++q)
        if (w[q] > w[big]) big = q;
    double sum = 0.0;
    for (int q = 0; q < 4; ++q)
        if (q != big) { w[q] = std::nearbyint(w[q] * 16777216.0) / 16777216.0; sum += w[q]; }
    w[big] = 1.0 - sum;
    // device order: (upwind v row, its side neighbour, own v row, its side neighbour)
    const int ord[4] = {2, 3, 0, 1};
    for (int q = 0; q < 4; ++q) rc.w[q] = (float)w[ord[q]];
    rc.kc = (float)(0.5 * r.ds);
    const double nrm = std::sqrt(r.mu[0] * r.mu[0] + r.mu[1] * r.mu[1] + r.mu[2] * r.mu[2]);
    for (int a = 0; a < 3; ++a) rc.mu[a] = (float)(r.mu[a] / nrm);
    rc.wq = (float)r.w;
    rc.active = 1;
    rc.up = r.up;
    rc.itop = r.itop;
}

void default_rays(rts_ctx* c)
{
    const double A = 0.2958759, B = 0.9082483;
    c->rays.clear();
    for (int o = 0; o < 8; ++o)
        for (int m = 0; m < 3; ++m) {
            HostRay r{};
            for (int a = 0; a < 3; ++a) {
                const double s = ((o >> a) & 1) ? -1.0 : 1.0;
                r.mu[a] = s * (a == m ? B : A);
            }
            r.w = 1.0 / 24.0;
            c->rays.push_back(r);
        }
}

// The sweep kernel is compiled for a few shared-memory row pitches (nodes per box row); a plan uses one.
constexpr int NPITCH = 4;
const int kPitch[NPITCH] = {24, 56, 72, 128};
const void* sweep_fn(int pitch, bool tolm = false)
{
    switch (pitch) {
        case 24: return tolm ? (const void*)tolp::rts_sweep_kernel<24> : (const void*)fixedp::rts_sweep_kernel<24>;
        case 56: return tolm ? (const void*)tolp::rts_sweep_kernel<56> : (const void*)fixedp::rts_sweep_kernel<56>;
        case 72: return tolm ? (const void*)tolp::rts_sweep_kernel<72> : (const void*)fixedp::rts_sweep_kernel<72>;
        default: return tolm ? (const void*)tolp::rts_sweep_kernel<128> : (const void*)fixedp::rts_sweep_kernel<128>;
    }
}
// dynamic shared memory of a CTA whose tiles are WU x WV (SmemPlan: coefficient ring, carried
// planes, ghost list, halo list)
int smem_for(int pitch, int WU, int WV, int ng, int nstage) { return (int)SmemPlan(pitch, WU, WV, ng, nstage).bytes(); }
// strips (node pair x rc rows, halo included, padded to whole warps) of ONE ray of a CTA whose tiles are
// WU x WV; a thread owns one
int items_for(int WU, int WV, int rc) { return SmemPlan::strips_for(WU, WV, rc); }

// --------------------------------------------------------------------------- planner
// Groups the rays into sweep units (march axis, direction, one ray per sign pair, band pair), chooses the
// tile shape, the ray groups per unit and the ring depth per march axis and the CTA size, lays out
// the workspace.
int make_plan(rts_ctx* c)
{
    c->planned = false;
    c->maps_ready = false;
    const int n[3] = {c->nx, c->ny, c->nz};
    int nup = 0;
    for (auto& r : c->rays) {
        if (ray_geometry(c->h, r) != 0) return fail(c, RTS_EINVAL, "ray with mu_z == 0");
        r.itop = r.up ? nup++ : -1;
    }
    c->n_up = nup;
    c->nbp = (c->nb + 1) / 2;
    for (int a = 0; a < 3; ++a) {
        TypePlan& t = c->tp[a];
        t.n_m = n[a];
        t.n_u = (a == 0) ? n[1] : n[0];
        t.n_v = (a == 2) ? n[1] : n[2];
    }
    c->PX = (int)align_up((size_t)c->nx, 4) + 2 * HALO;
    c->PY = (int)align_up((size_t)c->ny, 4) + 2 * HALO;
    c->PYR = c->ny + 2 * HALO;
    c->K = c->user_K ? c->user_K : KMAX;

    // --- unit skeletons: (march, dir) groups, sub-units with <= 1 ray per slot
    struct Group { int march, dir; std::vector<std::vector<int>> sub; };
    std::vector<Group> groups;
    for (int ri = 0; ri < (int)c->rays.size(); ++ri) {
        const HostRay& r = c->rays[ri];
        Group* g = nullptr;
        for (auto& gg : groups)
            if (gg.march == r.march && gg.dir == r.dir) g = &gg;
        if (!g) { groups.push_back(Group{r.march, r.dir, {}}); g = &groups.back(); }
        bool placed = false;
        for (auto& sub : g->sub) {
            bool freeslot = true;
            for (int rj : sub) freeslot &= (c->rays[rj].slot != r.slot);
            if (freeslot) { sub.push_back(ri); placed = true; break; }
        }
        if (!placed) g->sub.push_back(std::vector<int>{ri});
    }
    int skel_of[3] = {0, 0, 0};                  // (march, dir, sub) skeletons x band pairs
    for (auto& g : groups) skel_of[g.march] += (int)g.sub.size() * c->nbp;

    // --- per march axis: tile shape, ray groups per unit (2: all four rays of a plane in one CTA; 1: the
    //     su = +1 and su = -1 rays as separate units, for planes too large to be resident otherwise) and ring
    //     depth, by least modelled time among the shapes whose CTA fits R times on an SM
    cudaFuncAttributes fa;
    CUDA_TRY(c, cudaFuncGetAttributes(&fa, sweep_fn(56)));
    int bestR = 0, bestP = 0;
    double bestR_cost = 0.0;
    TypePlan best_tp[3];
    for (int R = (c->user_ctas_per_sm ? c->user_ctas_per_sm : 2); R >= 1; --R) {
      for (int pi = 0; pi < NPITCH; ++pi) {
        const int P = kPitch[pi];
        const int thread_cap = std::min(c->user_threads ? c->user_threads : RTS_SWEEP_THREADS, RTS_SWEEP_THREADS / R) / 128 * 128;
        const int smem_cap = std::min(c->max_smem_optin, (228 * 1024) / R - 1024 - (int)fa.sharedSizeBytes);
        const int slots = c->sm_count * R;
        bool ok = true;
        double costR = 0.0;
        TypePlan tp[3] = {c->tp[0], c->tp[1], c->tp[2]};
        for (int a = 0; a < 3 && ok; ++a) {
            TypePlan& t = tp[a];
            if (!skel_of[a]) { t.WU = 2; t.WV = 2; t.ntu = (t.n_u + 1) / 2; t.ntv = (t.n_v + 1) / 2; t.items = 0; t.ng = 2; t.nstage = 3; continue; }
            double best_cost = 0.0;
            int bu = 0, bv = 0, bng = 0, bns = 0;
            // rows per strip: as few row chunks as fit the thread budget (more rows per thread amortise the
            // per-step overhead), chunks of equal length
            auto rc_of = [&](int WU, int WV, int ng) {
                if (c->user_rc) return c->user_rc;
                const int nrows = WV + c->K - 1, npair = (WU + HALO) / 2;
                for (int nch = 1; nch <= nrows; ++nch) {
                    const int rc = (nrows + nch - 1) / nch;
                    if (rc <= 8 && 2 * ng * items_for(WU, WV, rc) <= thread_cap) return rc;
                }
                (void)npair;
                return 1;
            };
            const int n_u2 = (t.n_u + 1) & ~1;
            const int wu_max = std::min(n_u2, P - 2 * HALO);
            for (int ng = 2; ng >= 1; --ng) {
                if (c->user_ng && ng != c->user_ng) continue;
                for (int nst = 3; nst >= 2; --nst) {
                    if (c->user_nstage && nst != c->user_nstage) continue;
                    for (int WU = 2; WU <= wu_max; WU += 2) {
                        if (t.userWU && WU != std::min(wu_max, (t.userWU + 1) & ~1)) continue;
                        for (int WV = 1; WV <= std::min(t.n_v, 120); ++WV) {
                            if (t.userWV && WV != std::min(t.n_v, t.userWV)) continue;
                            if (smem_for(P, WU, WV, ng, nst) > smem_cap) break;
                            const int rc_try = rc_of(WU, WV, ng);
                            if (2 * ng * items_for(WU, WV, rc_try) > thread_cap) break;
                            const int ntu = (t.n_u + WU - 1) / WU, ntv = (t.n_v + WV - 1) / WV;
                            if ((long long)ntu * ntv > slots) continue;          // all tiles of a unit must be resident
                            // all tiles of a unit are resident together, so slots / ntiles units run at a time
                            const int uif = std::max(1, slots / (ntu * ntv));
                            const double units = (double)skel_of[a] * (2 / ng);
                            // ragged last tiles run at the pace of the full ones: charge the covered area
                            const double cover = ((double)ntu * WU * ntv * WV) / ((double)t.n_u * t.n_v);
                            // node-rays updated per step, averaged over a block: the u halo is a fixed strip while the
                            // v halo shrinks from K-1 rows to none; plus the per-step and per-block fixed costs and the
                            // box the TMA engine moves per step (the whole pitch, used or not)
                            const double work = 2.0 * ng * (WU + 0.75 * HALO) * (WV + 0.5 * (c->K - 1));
                            const double fixed = 700.0 + 6.0 * (WU + WV) + 0.25 * P * (WV + 2 * HALO);
                            double cost = units / uif * R * cover * (work + fixed);
                            if (nst == 2) cost *= 1.12;                          // the next plane's load is not hidden
                            // within the model's accuracy the tile that is wider along the unit-stride axis is taken
                            if (!bu || cost < 0.985 * best_cost || (cost < 1.015 * best_cost && ng == bng && nst == bns && WU > bu)) {
                                best_cost = cost; bu = WU; bv = WV; bng = ng; bns = nst;
                            }
                        }
                    }
                }
            }
            if (!bu) { ok = false; break; }
            t.WU = bu; t.WV = bv; t.ng = bng; t.nstage = bns;
            t.ntu = (t.n_u + bu - 1) / bu; t.ntv = (t.n_v + bv - 1) / bv;
            t.rc = rc_of(bu, bv, bng); t.items = items_for(bu, bv, t.rc);
            costR += best_cost;
        }
        if (ok && (!bestR || costR < 0.999 * bestR_cost)) { bestR = R; bestP = P; bestR_cost = costR; for (int a = 0; a < 3; ++a) best_tp[a] = tp[a]; }
      }
      if (c->user_ctas_per_sm) break;
    }
    if (bestR) for (int a = 0; a < 3; ++a) c->tp[a] = best_tp[a];
    if (!bestR) return fail(c, RTS_EINVAL, "planner: no tile shape fits (grid too large for one resident unit, or bad override)");
    c->pitch = bestP;
    c->smem_bytes = 0;
    c->threads = 64;
    for (int a = 0; a < 3; ++a)
        if (skel_of[a]) {
            const TypePlan& t = c->tp[a];
            c->smem_bytes = std::max(c->smem_bytes, smem_for(c->pitch, t.WU, t.WV, t.ng, t.nstage));
            c->threads = std::max(c->threads, 2 * t.ng * t.items);
        }
    c->threads = (c->threads + 127) / 128 * 128;               // two or four rays split the CTA into whole warps
    {
        int occ = 0;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, sweep_fn(c->pitch), c->threads, (size_t)c->smem_bytes) != cudaSuccess || occ < 1)
            return fail(c, RTS_ECUDA, "planner: sweep kernel does not fit on an SM");
        c->ctas_per_sm = std::min(bestR, occ);
    }
    const int slots = c->sm_count * c->ctas_per_sm;
    for (int a = 0; a < 3; ++a)
        if (skel_of[a] && c->tp[a].ntu * c->tp[a].ntv > slots)
            return fail(c, RTS_EINVAL, "planner: a sweep unit has more tiles than resident CTAs at the achieved occupancy");

    // --- materialise units in ticket order
    c->units.clear();
    int ticket = 0, uidx = 0;
    const size_t N = (size_t)c->nx * c->ny * c->nz;
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes, 256); return o; };
    const size_t fA = (size_t)c->nz * c->PYR * c->PX;          // nodes per field of layout A
    const size_t fB = (size_t)c->nz * c->nx * c->PY;
    c->off_coefA = take(sizeof(float2) * fA * 2 * c->nbp);
    c->off_coefB = take(sizeof(float2) * fB * 2 * c->nbp);
    c->nblk_a = ((c->nx + 31) / 32) * ((c->ny + 31) / 32);
    c->off_ksum = take(sizeof(double) * (size_t)c->nb * c->nz * c->nblk_a);
    c->off_kmin = take(sizeof(float) * (size_t)c->nb * c->nz * c->nblk_a);
    c->off_lev = take(sizeof(double) * (size_t)c->nb * c->nz * 2);
    c->off_kstar = take(sizeof(int) * c->nbp);
    c->off_mthick = take(sizeof(int) * c->nbp * 3);
    c->off_mthick_b = take(sizeof(int) * c->nb * 3);
    c->off_abort = take(sizeof(int) * 8);                    // [0] watchdog of the running launch, [1] ticket counter,
                                                             // [2] first watchdog code since the last rts_sync_check (sticky)
    for (auto& g : groups)
        for (auto& sub : g.sub)
            for (int b = 0; b < c->nbp; ++b) {
                const TypePlan& t = c->tp[g.march];
                for (int gi = 0; gi < (t.ng == 2 ? 1 : 2); ++gi) {     // one unit, or one per su
                    const int only_su = (t.ng == 2) ? 0 : (gi == 0 ? 1 : -1);
                    bool any = false;
                    for (int ri : sub) any |= (only_su == 0 || c->rays[ri].su == only_su);
                    if (!any) continue;
                    // band x octant sharding ("for N-bands ... run N times"): the units are
                    // dealt round robin to the ranks; a rank sweeps its own and leaves the others' heating at zero
                    if ((uidx++ % c->shard_n) != c->shard_rank) continue;
                    HostUnit hu{};
                    UnitDesc& d = hu.d;
                    std::memset(&d, 0, sizeof d);
                    d.march = g.march; d.dir = g.dir; d.pair = b;
                    d.per_v = (g.march == 2) ? 1 : 0;
                    d.n_m = t.n_m; d.n_u = t.n_u; d.n_v = t.n_v; d.n_u2 = (t.n_u + 1) & ~1;
                    d.WU = t.WU; d.WV = t.WV; d.ntu = t.ntu; d.ntv = t.ntv;
                    d.K = c->K; d.npass = c->npass;
                    d.ticket_begin = ticket;
                    d.ntiles = t.ntu * t.ntv;
                    ticket += d.ntiles;
                    d.nz = c->nz;
                    d.nstage = t.nstage; d.ng = t.ng; d.gsu0 = only_su ? only_su : 1; d.RC = t.rc;
                    d.nband_ok = (2 * b + 1 < c->nb) ? 2 : 1;
                    const long long nxy = (long long)c->nx * c->ny;
                    d.it_sr = nxy; d.it_sb = (long long)c->n_up * nxy;
                    if (g.march == 2)      { d.q_in_B = 0; d.q_sm = nxy;   d.q_sv = c->nx; d.it_su = 1;     d.it_so = c->nx; d.qvec = (c->nx % 2 == 0); }
                    else if (g.march == 1) { d.q_in_B = 0; d.q_sm = c->nx; d.q_sv = nxy;   d.it_su = 1;     d.it_so = c->nx; d.qvec = (c->nx % 2 == 0); }
                    else                   { d.q_in_B = 1; d.q_sm = c->ny; d.q_sv = nxy;   d.it_su = c->nx; d.it_so = 1;     d.qvec = (c->ny % 2 == 0); }
                    for (int q = 0; q < NSLOT; ++q) d.ray[q].itop = -1;
                    for (int ri : sub)
                        if (only_su == 0 || c->rays[ri].su == only_su) make_ray_consts(c->rays[ri], d.ray[c->rays[ri].slot]);
                    // tagged exchange: safe when every ray's strips are read by tiles whose own strips (of the opposite
                    // ray) this tile waits for before it writes the same buffer again (rts_sweep.cuh, block_start)
                    d.xflag = (t.ng == 2) ? 1 : 0;
                    for (int q = 0; q < NSLOT; ++q)
                        if (d.ray[q].active && !d.ray[q ^ 3].active) d.xflag = 0;
                    hu.off_xex = take(sizeof(float4) * 2 * NSLOT * (size_t)d.n_v * d.n_u2);
                    hu.off_g = take(sizeof(float2) * 2 * (size_t)d.n_m * NSLOT * (size_t)(d.n_v + d.n_u2));
                    hu.off_part = take(sizeof(float) * N * (c->flux ? 4 : 1));
                    hu.off_lp = (c->tol_max_passes > 0 && g.march != 2) ? take(sizeof(float2) * NSLOT * (size_t)d.n_v * d.n_u2) : 0;
                    c->units.push_back(hu);
                }
            }
    c->total_tickets = ticket;
    c->units_all = uidx;
    c->grid = std::min(slots, c->total_tickets);
    const size_t nu1 = std::max<size_t>(1, c->units.size());
    c->off_units = take(sizeof(UnitDesc) * nu1);
    c->off_partptr = take(sizeof(float*) * nu1);
    c->off_bar = take(sizeof(int) * nu1);
    c->off_errw = take(sizeof(unsigned) * nu1 * NSLOT * 4);
    c->off_stage_in = take(sizeof(float) * N * 3);
    c->off_stage_out = take(sizeof(float) * (N + (size_t)c->nb * c->n_up * c->ny * c->nx));
    c->ws_bytes = off;
    c->planned = true;
    return RTS_OK;
}

int bind_workspace(rts_ctx* c)
{
    unsigned char* ws = c->ws;
    std::vector<UnitDesc> flat;
    for (size_t i = 0; i < c->units.size(); ++i) {
        HostUnit& hu = c->units[i];
        UnitDesc& d = hu.d;
        d.Xex = (float*)(ws + hu.off_xex);
        d.Gu = (float*)(ws + hu.off_g);
        d.barrier = (int*)(ws + c->off_bar) + i;
        d.Qpart = (float*)(ws + hu.off_part);
        d.Fpart = c->flux ? d.Qpart + (size_t)c->nx * c->ny * c->nz : nullptr;
        d.Lp = (c->tol_max_passes > 0 && d.march != 2) ? (float*)(ws + hu.off_lp) : nullptr;
        d.errw = (unsigned*)(ws + c->off_errw) + i * NSLOT * 4;
        d.kstar = (const int*)(ws + c->off_kstar) + d.pair;
        d.mthick = (const int*)(ws + c->off_mthick) + 3 * d.pair;
        // exchange strips must not carry a stale tag and seam histories must be finite from the start (a skipped
        // thick plane copies its history from a carried plane that every task starts from zeros, and the exchange
        // strips of a skipped block are not read: nothing of an earlier solve reaches a later one)
        CUDA_TRY(c, cudaMemset(ws + hu.off_xex, 0, sizeof(float4) * 2 * NSLOT * (size_t)d.n_v * d.n_u2));
        CUDA_TRY(c, cudaMemset(ws + hu.off_g, 0, sizeof(float2) * 2 * (size_t)d.n_m * NSLOT * (size_t)(d.n_v + d.n_u2)));
        flat.push_back(d);
    }
    CUDA_TRY(c, cudaMemcpy(ws + c->off_units, flat.data(), sizeof(UnitDesc) * flat.size(), cudaMemcpyHostToDevice));
    {
        // the finalize kernel sums the x-fastest partials first (unit order), then the y-fastest ones (unit order)
        std::vector<float*> pp;
        for (auto& d : flat) if (!d.q_in_B) pp.push_back(d.Qpart);
        c->nplain = (int)pp.size();
        for (auto& d : flat) if (d.q_in_B) pp.push_back(d.Qpart);
        CUDA_TRY(c, cudaMemcpy(ws + c->off_partptr, pp.data(), sizeof(float*) * pp.size(), cudaMemcpyHostToDevice));
    }
    // coefficient tensors for the TMA engine (fp32 elements, two per node): layout A as (x, y rows, z, field)
    // with the box of the z-march (x, y) or of the y-march (x, z); layout B as (y, x, z, field) with the
    // x-march box (y, z)
    typedef CUresult (*EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                 const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                 CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    EncodeFn enc = (EncodeFn)c->encode_fn;
    for (int a = 0; a < 3; ++a) {
        const TypePlan& t = c->tp[a];
        const cuuint32_t BW = (cuuint32_t)(2 * c->pitch), BV = (cuuint32_t)(t.WV + 2 * HALO);
        // dimensions: (unit-stride axis, field, rows, planes, band pair); the box takes both fields of BV rows,
        // so a stage in shared memory is [BV][kaprho row | S row][pitch]
        cuuint64_t dims[5], strides[4];
        cuuint32_t box[5], estr[5] = {1, 1, 1, 1, 1};
        void* base;
        size_t fieldn;
        if (a == 0) {
            base = ws + c->off_coefB;
            fieldn = (size_t)c->nz * c->nx * c->PY;
            dims[0] = 2ull * c->PY; dims[2] = (cuuint64_t)c->nx; dims[3] = (cuuint64_t)c->nz;
            box[0] = BW; box[1] = 2; box[2] = 1; box[3] = BV; box[4] = 1;
        } else {
            base = ws + c->off_coefA;
            fieldn = (size_t)c->nz * c->PYR * c->PX;
            dims[0] = 2ull * c->PX; dims[2] = (cuuint64_t)c->PYR; dims[3] = (cuuint64_t)c->nz;
            if (a == 2) { box[0] = BW; box[1] = 2; box[2] = BV; box[3] = 1; box[4] = 1; }
            else        { box[0] = BW; box[1] = 2; box[2] = 1; box[3] = BV; box[4] = 1; }
        }
        dims[1] = 2; dims[4] = (cuuint64_t)c->nbp;
        strides[0] = fieldn * sizeof(float2);                   // field
        strides[1] = dims[0] * sizeof(float);                   // rows
        strides[2] = strides[1] * dims[2];                      // planes
        strides[3] = 2 * strides[0];                            // band pair
        CUresult r = enc(&c->maps.m[a], CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 5, base, dims, strides, box, estr,
                         CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                         CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) {
            char buf[96];
            snprintf(buf, sizeof buf, "cuTensorMapEncodeTiled failed (march %d, CUresult %d)", a, (int)r);
            return fail(c, RTS_ECUDA, buf);
        }
    }
    CUDA_TRY(c, cudaMemset(ws + c->off_abort, 0, sizeof(int) * 8));   // status word: a fresh workspace holds garbage
    c->pass_counter = 0;                                               // a fresh workspace holds no seam state
    c->maps_ready = true;
    return RTS_OK;
}

cudaStream_t as_stream(void* s) { return (cudaStream_t)s; }

int launch_stage_a(rts_ctx* c, const float* rho, const float* T, const float* P, float* plain_k, float* plain_s,
                   cudaStream_t st, int k0 = 0, int nk = -1)
{
    if (nk < 0) nk = c->nz;
    CoefParams p{};
    p.nx = c->nx; p.ny = c->ny; p.nz = c->nz; p.nb = c->nb; p.nT = c->nT; p.nP = c->nP;
    p.logT_min = c->logT_min; p.inv_dT = (c->nT - 1) / (c->logT_max - c->logT_min);
    p.logP_min = c->logP_min; p.inv_dP = (c->nP - 1) / (c->logP_max - c->logP_min);
    p.logkappa = c->d_logkappa; p.bandfrac = c->d_bandfrac;
    p.rho = rho; p.T = T; p.P = P;
    p.coefA = (float*)(c->ws + c->off_coefA); p.coefB = (float*)(c->ws + c->off_coefB);
    p.PX = c->PX; p.PY = c->PY; p.PYR = c->PYR;
    p.strideA_n = (long long)c->nz * c->PYR * c->PX;
    p.strideB_n = (long long)c->nz * c->nx * c->PY;
    p.ksum = (double*)(c->ws + c->off_ksum);
    p.kmin = (float*)(c->ws + c->off_kmin);
    p.plain_k = plain_k; p.plain_s = plain_s; p.k0 = k0;
    dim3 grid((c->nx + 31) / 32, (c->ny + 31) / 32, nk), block(32, 8);
    rts_coef_kernel<<<grid, block, 0, st>>>(p);
    CUDA_TRY(c, cudaGetLastError());
    return RTS_OK;
}

}  // namespace

// =========================================================================== C-ABI
extern "C" {

// Device address of g_scatter_scratch on device `dev`, which must be current; resolved once per device.
static cudaError_t resolve_static_scratch(int dev, void** ptr)
{
    static std::mutex mu;
    static struct { bool done; cudaError_t err; void* ptr; } tab[64] = {};
    if (dev < 0 || dev >= 64) { *ptr = nullptr; return cudaErrorInvalidDevice; }
    std::lock_guard<std::mutex> lock(mu);
    if (!tab[dev].done) {
        void* q = nullptr;
        tab[dev].err = cudaGetSymbolAddress(&q, g_scatter_scratch);
        tab[dev].ptr = (tab[dev].err == cudaSuccess) ? q : nullptr;
        tab[dev].done = true;
    }
    *ptr = tab[dev].ptr;
    return tab[dev].err;
}

int rts_create(rts_ctx** out, int nx, int ny, int nz, double dx, double dy, double dz, int nbands)
{
    if (!out) return RTS_EINVAL;
    *out = nullptr;
    if (nx < 2 || ny < 2 || nz < 2 || nbands < 1 || !(dx > 0) || !(dy > 0) || !(dz > 0))
        return fail(nullptr, RTS_EINVAL, "rts_create: need nx,ny,nz >= 2, nbands >= 1, positive spacings");
    if ((long long)nx * ny * nz > (1LL << 31) - 1) return fail(nullptr, RTS_EINVAL, "rts_create: grid too large");
    rts_ctx* c = new (std::nothrow) rts_ctx();
    if (!c) return RTS_ENOMEM;
    auto bail = [&](const std::string& m) { delete c; return fail(nullptr, RTS_ECUDA, "rts_create: " + m); };
    int dev = 0, ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev < 1) return bail(std::string("no CUDA device: ") + cudaGetErrorString(e));
    cudaDeviceProp prop;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess || (e = cudaGetDeviceProperties(&prop, dev)) != cudaSuccess)
        return bail(cudaGetErrorString(e));
    if (prop.major < 10) return bail("device is not sm_100: no other code path exists");
    int coop = 0;
    cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
    if (!coop) return bail("device lacks cooperative launch");
    c->sm_count = prop.multiProcessorCount;
    c->nx = nx; c->ny = ny; c->nz = nz; c->nb = nbands;
    c->h[0] = dx; c->h[1] = dy; c->h[2] = dz;
    default_rays(c);
    cudaFuncAttributes fa;
    if ((e = cudaFuncGetAttributes(&fa, sweep_fn(56))) != cudaSuccess) return bail(std::string("sweep kernel not loadable: ") + cudaGetErrorString(e));
    c->max_smem_optin = (int)prop.sharedMemPerBlockOptin - (int)fa.sharedSizeBytes;
    for (int pi = 0; pi < NPITCH; ++pi)
        for (int tm = 0; tm < 2; ++tm)
            if ((e = cudaFuncSetAttribute(sweep_fn(kPitch[pi], tm != 0), cudaFuncAttributeMaxDynamicSharedMemorySize, c->max_smem_optin)) != cudaSuccess)
                return bail(std::string("cudaFuncSetAttribute(max dynamic smem): ") + cudaGetErrorString(e));
    if ((e = cudaEventCreateWithFlags(&c->ev, cudaEventDisableTiming)) != cudaSuccess) return bail(cudaGetErrorString(e));
    {
        cudaDriverEntryPointQueryResult qres;
        if ((e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &c->encode_fn, cudaEnableDefault, &qres)) != cudaSuccess ||
            qres != cudaDriverEntryPointSuccess || !c->encode_fn)
            return bail("cuTensorMapEncodeTiled not available from the driver");
    }
    c->device = dev;
    c->static_scratch_err = resolve_static_scratch(dev, &c->static_scratch);   // reported by rts_scatter_solve_static only
    *out = c;
    return RTS_OK;
}

int rts_destroy(rts_ctx* c)
{
    if (!c) return RTS_EINVAL;
    if (c->d_logkappa) cudaFree(c->d_logkappa);
    if (c->d_bandfrac) cudaFree(c->d_bandfrac);
    if (c->ev) cudaEventDestroy(c->ev);
    for (auto& e : c->tev) if (e) cudaEventDestroy(e);
    for (auto& e : c->hev) if (e) cudaEventDestroy(e);
    if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
    delete c;
    return RTS_OK;
}

int rts_set_tables(rts_ctx* c, int nT, int nP, double logT_min, double logT_max, double logP_min,
                   double logP_max, const float* logkappa, const float* bandfrac)
{
    if (!c) return RTS_EINVAL;
    if (!logkappa || !bandfrac || nT < 2 || nP < 2 || !(logT_max > logT_min) || !(logP_max > logP_min))
        return fail(c, RTS_EINVAL, "rts_set_tables: bad argument");
    if (c->d_logkappa) { cudaFree(c->d_logkappa); c->d_logkappa = nullptr; }
    if (c->d_bandfrac) { cudaFree(c->d_bandfrac); c->d_bandfrac = nullptr; }
    c->have_tables = false;
    const size_t nk = (size_t)c->nb * nT * nP, nf = (size_t)c->nb * nT;
    CUDA_TRY(c, cudaMalloc(&c->d_logkappa, nk * sizeof(float)));
    CUDA_TRY(c, cudaMalloc(&c->d_bandfrac, nf * sizeof(float)));
    CUDA_TRY(c, cudaMemcpy(c->d_logkappa, logkappa, nk * sizeof(float), cudaMemcpyHostToDevice));
    CUDA_TRY(c, cudaMemcpy(c->d_bandfrac, bandfrac, nf * sizeof(float), cudaMemcpyHostToDevice));
    c->nT = nT; c->nP = nP;
    c->logT_min = logT_min; c->logT_max = logT_max; c->logP_min = logP_min; c->logP_max = logP_max;
    c->have_tables = true;
    return RTS_OK;
}

int rts_set_passes(rts_ctx* c, int npasses)
{
    if (!c) return RTS_EINVAL;
    if (npasses < 1) return fail(c, RTS_EINVAL, "rts_set_passes: npasses < 1");
    c->npass = npasses;
    c->planned = false;
    return RTS_OK;
}

int rts_set_rays(rts_ctx* c, int nrays, const double* mu, const double* w)
{
    if (!c) return RTS_EINVAL;
    if (!mu || !w || nrays < 1 || nrays > 256) return fail(c, RTS_EINVAL, "rts_set_rays: bad argument");
    std::vector<HostRay> rr;
    for (int r = 0; r < nrays; ++r) {
        HostRay h{};
        for (int a = 0; a < 3; ++a) h.mu[a] = mu[3 * r + a];
        if (h.mu[2] == 0.0 || !std::isfinite(h.mu[0]) || !std::isfinite(h.mu[1]) || !std::isfinite(h.mu[2]))
            return fail(c, RTS_EINVAL, "rts_set_rays: mu_z must be non-zero and finite");
        h.w = w[r];
        rr.push_back(h);
    }
    c->rays.swap(rr);
    c->planned = false;
    return RTS_OK;
}

int rts_get_rays(const rts_ctx* c, int* nrays, double* mu, double* w)
{
    if (!c || !nrays) return RTS_EINVAL;
    *nrays = (int)c->rays.size();
    for (size_t r = 0; r < c->rays.size(); ++r) {
        if (mu) for (int a = 0; a < 3; ++a) mu[3 * r + a] = c->rays[r].mu[a];
        if (w) w[r] = c->rays[r].w;
    }
    return RTS_OK;
}

int rts_num_up_rays(const rts_ctx* c)
{
    if (!c) return RTS_EINVAL;
    int n = 0;
    for (auto& r : c->rays) n += (r.mu[2] > 0.0);
    return n;
}

int rts_set_tiling(rts_ctx* c, int march, int tile_u, int tile_v)
{
    if (!c) return RTS_EINVAL;
    if (march < 0 || march > 2 || tile_u < 0 || tile_v < 0 || tile_u > 120 || tile_v > 120)
        return fail(c, RTS_EINVAL, "rts_set_tiling: bad argument");
    c->tp[march].userWU = tile_u;
    c->tp[march].userWV = tile_v;
    c->planned = false;
    return RTS_OK;
}

int rts_set_exchange_interval(rts_ctx* c, int k)
{
    if (!c) return RTS_EINVAL;
    if (k < 0 || k > KMAX) return fail(c, RTS_EINVAL, "rts_set_exchange_interval: 0..4");
    c->user_K = k;
    c->planned = false;
    return RTS_OK;
}

int rts_set_ring_depth(rts_ctx* c, int stages)
{
    if (!c) return RTS_EINVAL;
    if (stages != 0 && stages != 2 && stages != 3) return fail(c, RTS_EINVAL, "rts_set_ring_depth: 0, 2 or 3");
    c->user_nstage = stages;
    c->planned = false;
    return RTS_OK;
}

int rts_set_ctas_per_sm(rts_ctx* c, int n)
{
    if (!c) return RTS_EINVAL;
    if (n < 0 || n > 2) return fail(c, RTS_EINVAL, "rts_set_ctas_per_sm: 0..2");
    c->user_ctas_per_sm = n;
    c->planned = false;
    return RTS_OK;
}

size_t rts_workspace_bytes(rts_ctx* c)
{
    if (!c) return 0;
    if (!c->planned && make_plan(c) != RTS_OK) return 0;
    return c->ws_bytes;
}

int rts_set_workspace(rts_ctx* c, void* ws, size_t bytes)
{
    if (!c) return RTS_EINVAL;
    if (!c->planned) { int rc = make_plan(c); if (rc != RTS_OK) return rc; }
    if (!ws || ((uintptr_t)ws & 255u) != 0 || bytes < c->ws_bytes)
        return fail(c, RTS_EINVAL, "rts_set_workspace: null, misaligned or too small");
    c->ws = (unsigned char*)ws;
    c->ws_have = bytes;
    return bind_workspace(c);
}

int rts_plan_info(rts_ctx* c, int* what, int n)
{
    if (!c || !what) return RTS_EINVAL;
    if (!c->planned) { int rc = make_plan(c); if (rc != RTS_OK) return rc; }
    int zrays = 0;
    for (auto& r : c->rays) zrays += (r.march == 2);
    int v[16] = {4, c->total_tickets, c->ctas_per_sm, (int)c->units.size(), c->threads, c->smem_bytes,
                 c->grid, c->K, c->tp[0].WV, c->tp[1].WV, c->tp[2].WV, c->tp[0].WU, c->tp[1].WU, c->tp[2].WU,
                 zrays, c->units_all};
    for (int i = 0; i < n && i < 16; ++i) what[i] = v[i];
    return RTS_OK;
}

int rts_coefficients(rts_ctx* c, const float* rho, const float* T, const float* P, float* kaprho, float* S, void* stream)
{
    if (!c) return RTS_EINVAL;
    if (!rho || !T || !P || !kaprho || !S) return fail(c, RTS_EINVAL, "rts_coefficients: null pointer");
    if (!c->have_tables || !c->ws || !c->planned || !c->maps_ready) return fail(c, RTS_ESTATE, "rts_coefficients: tables/workspace not set");
    return launch_stage_a(c, rho, T, P, kaprho, S, as_stream(stream));
}

namespace {
int solve_impl(rts_ctx* c, const float* rho, const float* T, const float* P, float* Q, float* Itop,
               float* F, float* Qdiv, float* Qblend, void* stream, bool stage_a_done = false, cudaEvent_t after_sweep = nullptr)
{
    if (!c) return RTS_EINVAL;
    if (!rho || !T || !P || !Q) return fail(c, RTS_EINVAL, "rts_solve: null pointer");
    if (!c->have_tables) return fail(c, RTS_ESTATE, "rts_solve: tables not set");
    if (!c->ws || !c->planned || !c->maps_ready) return fail(c, RTS_ESTATE, "rts_solve: workspace not set (or configuration changed since)");
    if (((uintptr_t)Q & 15u) != 0) return fail(c, RTS_EINVAL, "rts_solve: Qrad must be 16-byte aligned");
    if ((F || Qdiv || Qblend) && !c->flux) return fail(c, RTS_ESTATE, "rts_solve_flux: call rts_enable_flux before sizing the workspace");
    if ((Qdiv || Qblend) && !F) return fail(c, RTS_EINVAL, "rts_solve_flux: Qdiv / Qblend need Frad");
    cudaStream_t st = as_stream(stream);
    const size_t N = (size_t)c->nx * c->ny * c->nz;
    unsigned char* ws = c->ws;

    // stage A + switch heights
    if (c->timing) CUDA_TRY(c, cudaEventRecord(c->tev[0], st));
    int rc = stage_a_done ? RTS_OK : launch_stage_a(c, rho, T, P, nullptr, nullptr, st);   // (rts_solve_host ran it slab by slab)
    if (rc != RTS_OK) return rc;
    {
        KstarParams kp{};
        kp.ksum = (const double*)(ws + c->off_ksum); kp.kmin = (const float*)(ws + c->off_kmin);
        kp.nb = c->nb; kp.nz = c->nz; kp.nblk = c->nblk_a;
        kp.inv_nxy = 1.0 / ((double)c->nx * c->ny); kp.dz = c->h[2]; kp.tau_switch = 5.0;
        for (int a = 0; a < 3; ++a) kp.kc[a] = 0.0;             // smallest half path of the rays marching along a (0: none)
        if (c->thick_skip)
            for (auto& r : c->rays) {
                const double k = (double)(float)(0.5 * r.ds);
                kp.kc[r.march] = (kp.kc[r.march] == 0.0) ? k : std::min(kp.kc[r.march], k);
            }
        kp.kstar_pair = (int*)(ws + c->off_kstar); kp.mthick_pair = (int*)(ws + c->off_mthick);
        kp.mthick_band = (int*)(ws + c->off_mthick_b); kp.lev = (double*)(ws + c->off_lev);
        rts_kstar_kernel<<<c->nbp, 1024, 0, st>>>(kp);             // 32 warps: the level sums are latency-bound loads
    }
    CUDA_TRY(c, cudaGetLastError());
    if (c->timing) CUDA_TRY(c, cudaEventRecord(c->tev[1], st));

    // the sweep: one persistent launch, tasks handed out by an in-order ticket counter.  Fixed pass count: one
    // launch runs all passes.  Error-controlled mode (NEXT #3): one pass per launch; after each the host reads the
    // units' error words and stops when the seam faces of every (band, ray) changed by <= tol * max|I| on them.
    if (c->timing) CUDA_TRY(c, cudaEventRecord(c->tev[2], st));
    if (c->shard_n > 1 && Itop)    // the emergent intensities of the other ranks' rays stay zero: a sum over ranks completes them
        CUDA_TRY(c, cudaMemsetAsync(Itop, 0, sizeof(float) * (size_t)c->nb * c->n_up * c->ny * c->nx, st));
    const bool tolmode = c->tol_max_passes > 0;
    if (tolmode && !c->warm) c->pass_counter = 0;
    const int nlaunch = tolmode ? c->tol_max_passes : 1;
    c->passes_used = 0;
    for (int it = 0; it < nlaunch && c->total_tickets > 0; ++it) {
        CUDA_TRY(c, cudaMemsetAsync(ws + c->off_abort, 0, sizeof(int) * 2, st));   // not the sticky word
        CUDA_TRY(c, cudaMemsetAsync(ws + c->off_bar, 0, sizeof(int) * c->units.size(), st));
        if (tolmode) CUDA_TRY(c, cudaMemsetAsync(ws + c->off_errw, 0, sizeof(unsigned) * c->units.size() * NSLOT * 4, st));
        const UnitDesc* dunits = (const UnitDesc*)(ws + c->off_units);
        int* abortf = (int*)(ws + c->off_abort);
        int* ticket = abortf + 1;
        int nunits = (int)c->units.size(), total = c->total_tickets;
        unsigned seq = ++c->solve_seq;                          // tags of this launch's exchange words
        if ((seq & 0xfffffu) == 0) seq = ++c->solve_seq;
        seq &= 0xfffffu;
        int pbase = tolmode ? c->pass_counter : 0, npl = tolmode ? 1 : 0;
        void* args[] = {&c->maps, &dunits, &nunits, &total, &ticket, &Itop, &abortf, &seq, &pbase, &npl};
        // cooperative launch: every CTA of the grid is resident, which the tile barriers rely on
        CUDA_TRY(c, cudaLaunchCooperativeKernel(sweep_fn(c->pitch, tolmode), dim3(c->grid), dim3(c->threads), args,
                                                (size_t)c->smem_bytes, st));
        if (!tolmode) break;
        ++c->pass_counter; ++c->passes_used;
        std::vector<unsigned> ew(c->units.size() * NSLOT * 4);
        CUDA_TRY(c, cudaMemcpyAsync(ew.data(), ws + c->off_errw, sizeof(unsigned) * ew.size(), cudaMemcpyDeviceToHost, st));
        CUDA_TRY(c, cudaStreamSynchronize(st));
        float worst = 0.f;
        for (size_t q = 0; q < ew.size(); q += 4)
            for (int b = 0; b < 2; ++b) {
                float e, sc;
                std::memcpy(&e, &ew[q + b], 4); std::memcpy(&sc, &ew[q + 2 + b], 4);
                if (sc > 0.f) worst = std::max(worst, e / sc);
            }
        c->relerr_last = worst;
        if ((double)worst <= c->tol) break;
    }
    // finalize
    if (c->timing) CUDA_TRY(c, cudaEventRecord(c->tev[3], st));
    if (after_sweep) CUDA_TRY(c, cudaEventRecord(after_sweep, st));
    {
        // the units' partial heating (and flux) summed in unit order: deterministic
        FinalizeParams fp{};
        fp.part = (const float* const*)(ws + c->off_partptr); fp.nplain = c->nplain;
        fp.nunits = (int)c->units.size(); fp.nf = F ? 4 : 1;
        fp.nx = c->nx; fp.ny = c->ny; fp.nz = c->nz;
        fp.out[0] = Q;
        for (int a = 0; a < 3; ++a) fp.out[1 + a] = F ? F + (size_t)a * N : nullptr;
        dim3 grid((c->nx + 31) / 32, (c->ny + 31) / 32, c->nz), block(32, 8);
        rts_finalize_kernel<<<grid, block, 0, st>>>(fp);
        CUDA_TRY(c, cudaGetLastError());
        if (Qdiv || Qblend) {
            dim3 g2((c->nx + 255) / 256, c->ny, c->nz);
            rts_fluxdiv_kernel<<<g2, 256, 0, st>>>(F, Q, Qdiv, Qblend, (const double*)(ws + c->off_lev), c->nx, c->ny, c->nz,
                                                   (float)c->h[0], (float)c->h[1], (float)c->h[2],
                                                   1.0 / ((double)c->nx * c->ny), c->h[2], c->tau0);
            CUDA_TRY(c, cudaGetLastError());
        }
    }
    if (c->timing) CUDA_TRY(c, cudaEventRecord(c->tev[4], st));
    return RTS_OK;
}
}  // namespace

int rts_solve(rts_ctx* c, const float* rho, const float* T, const float* P, float* Q, float* Itop, void* stream)
{
    return solve_impl(c, rho, T, P, Q, Itop, nullptr, nullptr, nullptr, stream);
}

int rts_enable_flux(rts_ctx* c, int on)
{
    if (!c) return RTS_EINVAL;
    c->flux = on != 0;
    c->planned = false;
    return RTS_OK;
}

int rts_set_flux_blend(rts_ctx* c, double tau0)
{
    if (!c) return RTS_EINVAL;
    if (!(tau0 > 0.0)) return fail(c, RTS_EINVAL, "rts_set_flux_blend: tau0 must be positive");
    c->tau0 = tau0;
    return RTS_OK;
}

int rts_solve_flux(rts_ctx* c, const float* rho, const float* T, const float* P, float* Q, float* Itop,
                   float* Frad, float* Qdiv, float* Qblend, void* stream)
{
    if (!c) return RTS_EINVAL;
    if (!Frad) return fail(c, RTS_EINVAL, "rts_solve_flux: null Frad");
    return solve_impl(c, rho, T, P, Q, Itop, Frad, Qdiv, Qblend, stream);
}

int rts_set_tolerance(rts_ctx* c, double tol, int max_passes)
{
    if (!c) return RTS_EINVAL;
    if (max_passes < 0 || max_passes > 4096 || !(tol == tol)) return fail(c, RTS_EINVAL, "rts_set_tolerance: 0 <= max_passes <= 4096, tol not NaN");
    const bool was = c->tol_max_passes > 0, is = max_passes > 0;
    c->tol = tol; c->tol_max_passes = max_passes;
    if (was != is) c->planned = false;             // the last-plane buffers exist in this mode only
    c->pass_counter = 0;
    return RTS_OK;
}

int rts_set_warm_start(rts_ctx* c, int on)
{
    if (!c) return RTS_EINVAL;
    c->warm = on != 0;
    if (!c->warm) c->pass_counter = 0;
    return RTS_OK;
}

int rts_passes_used(rts_ctx* c, int* passes, float* relerr_last)
{
    if (!c) return RTS_EINVAL;
    if (c->tol_max_passes <= 0) return fail(c, RTS_ESTATE, "rts_passes_used: error-controlled mode is off (rts_set_tolerance)");
    if (passes) *passes = c->passes_used;
    if (relerr_last) *relerr_last = c->relerr_last;
    return RTS_OK;
}

int rts_set_shard(rts_ctx* c, int rank, int nranks)
{
    if (!c) return RTS_EINVAL;
    if (nranks < 1 || rank < 0 || rank >= nranks) return fail(c, RTS_EINVAL, "rts_set_shard: need 0 <= rank < nranks");
    c->shard_rank = rank; c->shard_n = nranks;
    c->planned = false;
    return RTS_OK;
}

int rts_shard_info(rts_ctx* c, int* units_mine, int* units_all)
{
    if (!c) return RTS_EINVAL;
    if (!c->planned) { int rc = make_plan(c); if (rc != RTS_OK) return rc; }
    if (units_mine) *units_mine = (int)c->units.size();
    if (units_all) *units_all = c->units_all;
    return RTS_OK;
}

int rts_set_thick_skip(rts_ctx* c, int on)
{
    if (!c) return RTS_EINVAL;
    c->thick_skip = on != 0;
    return RTS_OK;
}

int rts_thick_levels(rts_ctx* c, int* levels_host, void* stream)
{
    if (!c || !levels_host) return RTS_EINVAL;
    if (!c->ws || !c->planned) return fail(c, RTS_ESTATE, "rts_thick_levels: workspace not set");
    CUDA_TRY(c, cudaStreamSynchronize(as_stream(stream)));
    std::vector<int> lv((size_t)c->nb * 3);
    CUDA_TRY(c, cudaMemcpy(lv.data(), c->ws + c->off_mthick_b, sizeof(int) * lv.size(), cudaMemcpyDeviceToHost));
    for (int b = 0; b < c->nb; ++b) levels_host[b] = lv[(size_t)b * 3 + 2];
    return RTS_OK;
}

int rts_enable_timing(rts_ctx* c, int on)
{
    if (!c) return RTS_EINVAL;
    if (on) for (auto& e : c->tev) if (!e) CUDA_TRY(c, cudaEventCreate(&e));
    c->timing = on != 0;
    return RTS_OK;
}

int rts_last_timing(rts_ctx* c, float* ms4)
{
    if (!c || !ms4) return RTS_EINVAL;
    if (!c->timing) return fail(c, RTS_ESTATE, "rts_last_timing: timing not enabled");
    CUDA_TRY(c, cudaEventSynchronize(c->tev[4]));
    CUDA_TRY(c, cudaEventElapsedTime(&ms4[0], c->tev[0], c->tev[1]));
    CUDA_TRY(c, cudaEventElapsedTime(&ms4[1], c->tev[2], c->tev[3]));
    CUDA_TRY(c, cudaEventElapsedTime(&ms4[2], c->tev[3], c->tev[4]));
    CUDA_TRY(c, cudaEventElapsedTime(&ms4[3], c->tev[0], c->tev[4]));
    return RTS_OK;
}

int rts_sync_check(rts_ctx* c, void* stream)
{
    if (!c) return RTS_EINVAL;
    cudaError_t e = cudaStreamSynchronize(as_stream(stream));
    if (e != cudaSuccess) return fail(c, RTS_ECUDA, std::string("stream sync: ") + cudaGetErrorString(e));
    if (c->ws) {
        // the sticky word: a watchdog that fired in any solve queued since the last check is reported, not only the
        // last solve's (every solve clears the word its own launches test)
        int ab = 0;
        e = cudaMemcpy(&ab, c->ws + c->off_abort + 2 * sizeof(int), sizeof(int), cudaMemcpyDeviceToHost);
        if (e != cudaSuccess) return fail(c, RTS_ECUDA, std::string("status read: ") + cudaGetErrorString(e));
        if (ab) {
            cudaMemset(c->ws + c->off_abort + 2 * sizeof(int), 0, sizeof(int));
            char buf[256];
            snprintf(buf, sizeof buf, "sweep kernel watchdog fired (code %d, step %d): a wait did not complete", ab & 15, ab >> 4);
            return fail(c, RTS_ETIMEOUT, buf);
        }
    }
    return RTS_OK;
}

int rts_solve_host(rts_ctx* c, const float* rho, const float* T, const float* P, float* Q, float* Itop, void* stream)
{
    if (!c) return RTS_EINVAL;
    if (!rho || !T || !P || !Q) return fail(c, RTS_EINVAL, "rts_solve_host: null pointer");
    if (!c->ws || !c->planned || !c->maps_ready) return fail(c, RTS_ESTATE, "rts_solve_host: workspace not set");
    cudaStream_t st = as_stream(stream);
    const size_t N = (size_t)c->nx * c->ny * c->nz;
    const size_t nI = (size_t)c->nb * c->n_up * c->ny * c->nx;
    float* din = (float*)(c->ws + c->off_stage_in);
    float* dout = (float*)(c->ws + c->off_stage_out);
    // Copies and kernels overlap: rho, T, P arrive in slabs of levels on a second stream, stage A follows slab by
    // slab on the caller's stream; I_top goes back while the finalize kernel runs.
    if (!c->copy_stream) {
        CUDA_TRY(c, cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking));
        for (auto& e : c->hev) CUDA_TRY(c, cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    }
    constexpr int NSLAB = 8;
    CUDA_TRY(c, cudaEventRecord(c->hev[NSLAB], st));                      // earlier work on the caller's stream still reads din
    CUDA_TRY(c, cudaStreamWaitEvent(c->copy_stream, c->hev[NSLAB], 0));
    const size_t plane = (size_t)c->nx * c->ny;
    for (int sl = 0; sl < NSLAB; ++sl) {
        const int k0 = (int)((long long)c->nz * sl / NSLAB), k1 = (int)((long long)c->nz * (sl + 1) / NSLAB);
        if (k1 <= k0) continue;
        const size_t o = plane * k0, n = plane * (k1 - k0) * sizeof(float);
        CUDA_TRY(c, cudaMemcpyAsync(din + o, rho + o, n, cudaMemcpyHostToDevice, c->copy_stream));
        CUDA_TRY(c, cudaMemcpyAsync(din + N + o, T + o, n, cudaMemcpyHostToDevice, c->copy_stream));
        CUDA_TRY(c, cudaMemcpyAsync(din + 2 * N + o, P + o, n, cudaMemcpyHostToDevice, c->copy_stream));
        CUDA_TRY(c, cudaEventRecord(c->hev[sl], c->copy_stream));
        CUDA_TRY(c, cudaStreamWaitEvent(st, c->hev[sl], 0));
        if (!c->have_tables) return fail(c, RTS_ESTATE, "rts_solve_host: tables not set");
        int rcA = launch_stage_a(c, din, din + N, din + 2 * N, nullptr, nullptr, st, k0, k1 - k0);
        if (rcA != RTS_OK) return rcA;
    }
    int rc = solve_impl(c, din, din + N, din + 2 * N, dout, Itop ? dout + N : nullptr, nullptr, nullptr, nullptr, stream,
                        true, c->hev[NSLAB + 1]);
    if (rc != RTS_OK) return rc;
    if (Itop && c->tol_max_passes <= 0) {
        CUDA_TRY(c, cudaStreamWaitEvent(c->copy_stream, c->hev[NSLAB + 1], 0));
        CUDA_TRY(c, cudaMemcpyAsync(Itop, dout + N, nI * sizeof(float), cudaMemcpyDeviceToHost, c->copy_stream));
    } else if (Itop) {
        CUDA_TRY(c, cudaMemcpyAsync(Itop, dout + N, nI * sizeof(float), cudaMemcpyDeviceToHost, st));
    }
    CUDA_TRY(c, cudaMemcpyAsync(Q, dout, N * sizeof(float), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(c, cudaStreamSynchronize(c->copy_stream));
    return rts_sync_check(c, stream);
}

namespace {
int launch_c2n(rts_ctx* c, int nf, const float* const* cell, float* const* node, cudaStream_t st)
{
    StaggerParams p{};
    p.nx = c->nx; p.ny = c->ny; p.nz = c->nz; p.nf = nf; p.zchunk = 32;
    for (int f = 0; f < nf; ++f) { p.cell[f] = cell[f]; p.node[f] = node[f]; }
    dim3 block(64, 4), grid((c->nx + 63) / 64, (c->ny + 3) / 4, (c->nz + p.zchunk - 1) / p.zchunk);
    rts_cells_to_nodes_kernel<<<grid, block, 0, st>>>(p);
    CUDA_TRY(c, cudaGetLastError());
    return RTS_OK;
}
int launch_n2c(rts_ctx* c, const float* qn, float* qc, cudaStream_t st)
{
    const int zchunk = 32;
    dim3 block(64, 4), grid((c->nx + 63) / 64, (c->ny + 3) / 4, (c->nz - 1 + zchunk - 1) / zchunk);
    rts_nodes_to_cells_kernel<<<grid, block, 0, st>>>(qn, qc, c->nx, c->ny, c->nz, zchunk);
    CUDA_TRY(c, cudaGetLastError());
    return RTS_OK;
}
}  // namespace

int rts_cells_to_nodes(rts_ctx* c, const float* cell, float* node, void* stream)
{
    if (!c) return RTS_EINVAL;
    if (!cell || !node) return fail(c, RTS_EINVAL, "rts_cells_to_nodes: null pointer");
    return launch_c2n(c, 1, &cell, &node, as_stream(stream));
}

int rts_nodes_to_cells(rts_ctx* c, const float* qn, float* qc, void* stream)
{
    if (!c) return RTS_EINVAL;
    if (!qn || !qc) return fail(c, RTS_EINVAL, "rts_nodes_to_cells: null pointer");
    return launch_n2c(c, qn, qc, as_stream(stream));
}

int rts_solve_cells(rts_ctx* c, const float* rho_c, const float* T_c, const float* P_c, float* Qc, float* Itop, void* stream)
{
    if (!c) return RTS_EINVAL;
    if (!rho_c || !T_c || !P_c || !Qc) return fail(c, RTS_EINVAL, "rts_solve_cells: null pointer");
    if (!c->ws || !c->planned || !c->maps_ready) return fail(c, RTS_ESTATE, "rts_solve_cells: workspace not set");
    const size_t N = (size_t)c->nx * c->ny * c->nz;
    float* din = (float*)(c->ws + c->off_stage_in);      // node fields rho, T, P
    float* qn = (float*)(c->ws + c->off_stage_out);      // node heating
    const float* cell[3] = {rho_c, T_c, P_c};
    float* node[3] = {din, din + N, din + 2 * N};
    int rc = launch_c2n(c, 3, cell, node, as_stream(stream));
    if (rc != RTS_OK) return rc;
    rc = rts_solve(c, din, din + N, din + 2 * N, qn, Itop, stream);
    if (rc != RTS_OK) return rc;
    return launch_n2c(c, qn, Qc, as_stream(stream));
}

// ---- scattering source function, source update along the ray (NEXT #4; rts_scatter.cuh)
static size_t scatter_layout(const rts_ctx* c, int nbands, int niter, size_t off[8])
{
    const size_t N = (size_t)c->nx * c->ny * c->nz, nr = c->rays.size(), nb = (size_t)nbands;
    size_t o = 0;
    auto take = [&](size_t bytes) { size_t r = o; o = align_up(o + bytes, 256); return r; };
    off[0] = take(sizeof(double) * N * nr * nb);                 // I_r of every band
    off[1] = take(sizeof(double) * (size_t)c->nz * c->ny * nb);  // faceX
    off[2] = take(sizeof(double) * (size_t)c->nz * c->nx * nb);  // faceY
    off[3] = take(sizeof(double) * N * nb);                      // S of the previous iteration
    off[4] = take(sizeof(ScatRay) * nr);
    off[5] = take(sizeof(unsigned long long) * 2 * nb * (size_t)std::max(niter, 1));
    off[6] = take(sizeof(unsigned) * 4);
    off[7] = take(sizeof(float) * 3 * N * nb);                   // y-fastest copies of kaprho, B, eps
    return o;
}

size_t rts_scatter_workspace_bytes(rts_ctx* c, int nbands, int niter)
{
    if (!c || nbands < 1 || nbands > 1024 || niter < 0 || niter > 65536) return 0;
    size_t off[8];
    return scatter_layout(c, nbands, niter, off);
}

int rts_scatter_solve(rts_ctx* c, int nbands, const float* kaprho, const float* B, const float* eps, int niter, int gauss_seidel,
                      void* workspace, size_t ws_bytes, double* S, double* J, double* change_host, void* stream)
{
    if (!c) return RTS_EINVAL;
    if (!kaprho || !B || !eps || !S || !J || !workspace) return fail(c, RTS_EINVAL, "rts_scatter_solve: null pointer");
    if (niter < 0 || niter > 65536 || nbands < 1 || nbands > 1024) return fail(c, RTS_EINVAL, "rts_scatter_solve: 0 <= niter <= 65536, 1 <= nbands <= 1024");
    size_t off[8];
    const size_t need = scatter_layout(c, nbands, niter, off);
    if (((uintptr_t)workspace & 255u) != 0 || ws_bytes < need) return fail(c, RTS_EINVAL, "rts_scatter_solve: workspace misaligned or too small");
    cudaStream_t st = as_stream(stream);
    unsigned char* ws = (unsigned char*)workspace;
    // ray geometry (reading R3) in node offsets
    c->scat_rays.clear();
    for (HostRay r : c->rays) {
        if (ray_geometry(c->h, r) != 0) return fail(c, RTS_EINVAL, "ray with mu_z == 0");
        ScatRay q{};
        const int as = r.march, ua = (as == 0) ? 1 : 0, va = (as == 2) ? 1 : 2;
        q.as = as; q.dir = r.dir; q.up = r.up; q.kdir = r.up ? 0 : c->nz - 1;
        int sg[3]; sg[as] = r.dir; sg[ua] = r.su; sg[va] = r.sv;
        q.iface = (sg[0] > 0) ? c->nx - 1 : 0; q.jface = (sg[1] > 0) ? c->ny - 1 : 0;
        for (int eu = 0; eu < 2; ++eu)
            for (int ev = 0; ev < 2; ++ev) {
                const int t = eu * 2 + ev;
                q.off[t][0] = q.off[t][1] = q.off[t][2] = 0;
                q.off[t][as] = -sg[as]; q.off[t][ua] = -eu * sg[ua]; q.off[t][va] = -ev * sg[va];
                q.w[t] = (eu ? r.fu : 1.0 - r.fu) * (ev ? r.fv : 1.0 - r.fv);
            }
        q.ds = r.ds; q.wq = r.w;
        c->scat_rays.push_back(q);
    }
    CUDA_TRY(c, cudaMemcpyAsync(ws + off[4], c->scat_rays.data(), sizeof(ScatRay) * c->scat_rays.size(), cudaMemcpyHostToDevice, st));
    CUDA_TRY(c, cudaMemsetAsync(ws + off[5], 0, sizeof(unsigned long long) * 2 * (size_t)nbands * (size_t)std::max(niter, 1), st));
    CUDA_TRY(c, cudaMemsetAsync(ws + off[6], 0, sizeof(unsigned) * 4, st));
    ScatParams p{};
    p.nx = c->nx; p.ny = c->ny; p.nz = c->nz; p.nrays = (int)c->rays.size(); p.niter = niter; p.gs = gauss_seidel != 0; p.nb = nbands;
    p.kaprho = kaprho; p.B = B; p.eps = eps;
    p.rays = (const ScatRay*)(ws + off[4]);
    p.I = (double*)(ws + off[0]); p.faceX = (double*)(ws + off[1]); p.faceY = (double*)(ws + off[2]); p.Sold = (double*)(ws + off[3]);
    p.S = S; p.J = J;
    p.chg = (unsigned long long*)(ws + off[5]); p.bar = (unsigned*)(ws + off[6]);
    { const size_t NBn = (size_t)c->nx * c->ny * c->nz * (size_t)nbands; p.kapT = (float*)(ws + off[7]); p.BT = p.kapT + NBn; p.epsT = p.BT + NBn; }
    const size_t plane_max = (size_t)std::max(c->nx, c->ny) * std::max(std::max(c->nx, c->ny), c->nz);
    // the variant with 3 CTAs per SM where 2 per SM would leave some threads with a second node per plane step
    const bool big = plane_max * nbands > (size_t)c->sm_count * 2 * 256;
    const void* kern = big ? (const void*)rts_scatter_kernel<3> : (const void*)rts_scatter_kernel<2>;
    int occ = 0;
    CUDA_TRY(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, 256, 0));
    if (occ < 1) return fail(c, RTS_ECUDA, "rts_scatter_solve: kernel does not fit on an SM");
    const int grid = (int)std::max<size_t>(1, std::min<size_t>((size_t)c->sm_count * std::min(occ, 4), (plane_max * nbands + 255) / 256));
    void* args[] = {&p};
    // cooperative launch: every CTA is resident, which the grid-wide barrier between planes relies on
    CUDA_TRY(c, cudaLaunchCooperativeKernel(kern, dim3(grid), dim3(256), args, 0, st));
    std::vector<unsigned long long> chg(2 * (size_t)nbands * (size_t)std::max(niter, 1));
    unsigned flags[4] = {0, 0, 0, 0};
    CUDA_TRY(c, cudaMemcpyAsync(chg.data(), ws + off[5], sizeof(unsigned long long) * chg.size(), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(c, cudaMemcpyAsync(flags, ws + off[6], sizeof(flags), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(c, cudaStreamSynchronize(st));
    if (flags[1] != 0) return fail(c, RTS_ETIMEOUT, "rts_scatter_solve: the grid barrier timed out");
    if (change_host)
        for (size_t q = 0; q < (size_t)niter * nbands; ++q) {                 // [niter][nbands]
            double e, sc;
            std::memcpy(&e, &chg[2 * q], 8); std::memcpy(&sc, &chg[2 * q + 1], 8);
            change_host[q] = (sc > 0.0) ? e / sc : 0.0;
        }
    return RTS_OK;
}

// The same solve with its scratch in the static device array: allocates nothing (no cudaMalloc / cudaFree, no host
// heap: the ray constants and the change words live on the stack, which bounds nrays and niter * nbands).
int rts_scatter_solve_static(rts_ctx* c, int nbands, const float* kaprho, const float* B, const float* eps, int niter,
                             int gauss_seidel, double* S, double* J, double* change_host, void* stream)
{
    constexpr int MAXR = 256, MAXCHG = 2048;
    if (!c) return RTS_EINVAL;
    if (!kaprho || !B || !eps || !S || !J) return fail(c, RTS_EINVAL, "rts_scatter_solve_static: null pointer");
    if (niter < 0 || nbands < 1 || (long long)std::max(niter, 1) * nbands > MAXCHG)
        return fail(c, RTS_EINVAL, "rts_scatter_solve_static: need niter >= 0, nbands >= 1, max(niter, 1) * nbands <= 2048");
    const int nr = (int)c->rays.size();
    if (nr < 1 || nr > MAXR) return fail(c, RTS_EINVAL, "rts_scatter_solve_static: 1 <= rays <= 256");
    int dev = -1;
    CUDA_TRY(c, cudaGetDevice(&dev));
    if (dev != c->device) return fail(c, RTS_ESTATE, "rts_scatter_solve_static: the context's device is not current");
    if (c->static_scratch_err != cudaSuccess || !c->static_scratch)
        return fail(c, RTS_ECUDA, std::string("rts_scatter_solve_static: cudaGetSymbolAddress of the static scratch failed at set-up: ") +
                                      cudaGetErrorString(c->static_scratch_err));
    size_t off[8];
    const size_t need = scatter_layout(c, nbands, niter, off);
    if (need > (size_t)RTS_SCATTER_STATIC_BYTES_IMPL) {
        char buf[200];
        snprintf(buf, sizeof buf, "rts_scatter_solve_static: this problem needs %zu bytes of scratch, the static array holds %u "
                                  "(use rts_scatter_solve with a caller-owned workspace)", need, (unsigned)RTS_SCATTER_STATIC_BYTES_IMPL);
        return fail(c, RTS_EINVAL, buf);
    }
    cudaStream_t st = as_stream(stream);
    unsigned char* ws = (unsigned char*)c->static_scratch;       // the DEVICE address, never the symbol's name
    ScatRay rays[MAXR];
    for (int i = 0; i < nr; ++i) {
        HostRay r = c->rays[i];
        if (ray_geometry(c->h, r) != 0) return fail(c, RTS_EINVAL, "ray with mu_z == 0");
        ScatRay q{};
        const int as = r.march, ua = (as == 0) ? 1 : 0, va = (as == 2) ? 1 : 2;
        q.as = as; q.dir = r.dir; q.up = r.up; q.kdir = r.up ? 0 : c->nz - 1;
        int sg[3]; sg[as] = r.dir; sg[ua] = r.su; sg[va] = r.sv;
        q.iface = (sg[0] > 0) ? c->nx - 1 : 0; q.jface = (sg[1] > 0) ? c->ny - 1 : 0;
        for (int eu = 0; eu < 2; ++eu)
            for (int ev = 0; ev < 2; ++ev) {
                const int t = eu * 2 + ev;
                q.off[t][0] = q.off[t][1] = q.off[t][2] = 0;
                q.off[t][as] = -sg[as]; q.off[t][ua] = -eu * sg[ua]; q.off[t][va] = -ev * sg[va];
                q.w[t] = (eu ? r.fu : 1.0 - r.fu) * (ev ? r.fv : 1.0 - r.fv);
            }
        q.ds = r.ds; q.wq = r.w;
        rays[i] = q;
    }
    const size_t nchg = 2 * (size_t)nbands * (size_t)std::max(niter, 1);
    // the array keeps the previous call's contents: the change words and the barrier words must start at zero (the
    // kernel itself initialises I_r, J, S and rewrites the faces and S_old before it reads them)
    CUDA_TRY(c, cudaMemcpyAsync(ws + off[4], rays, sizeof(ScatRay) * nr, cudaMemcpyHostToDevice, st));
    CUDA_TRY(c, cudaMemsetAsync(ws + off[5], 0, sizeof(unsigned long long) * nchg, st));
    CUDA_TRY(c, cudaMemsetAsync(ws + off[6], 0, sizeof(unsigned) * 4, st));
    ScatParams p{};
    p.nx = c->nx; p.ny = c->ny; p.nz = c->nz; p.nrays = nr; p.niter = niter; p.gs = gauss_seidel != 0; p.nb = nbands;
    p.kaprho = kaprho; p.B = B; p.eps = eps;
    p.rays = (const ScatRay*)(ws + off[4]);
    p.I = (double*)(ws + off[0]); p.faceX = (double*)(ws + off[1]); p.faceY = (double*)(ws + off[2]); p.Sold = (double*)(ws + off[3]);
    p.S = S; p.J = J;
    p.chg = (unsigned long long*)(ws + off[5]); p.bar = (unsigned*)(ws + off[6]);
    { const size_t NBn = (size_t)c->nx * c->ny * c->nz * (size_t)nbands; p.kapT = (float*)(ws + off[7]); p.BT = p.kapT + NBn; p.epsT = p.BT + NBn; }
    const size_t plane_max = (size_t)std::max(c->nx, c->ny) * std::max(std::max(c->nx, c->ny), c->nz);
    // the variant with 3 CTAs per SM where 2 per SM would leave some threads with a second node per plane step
    const bool big = plane_max * nbands > (size_t)c->sm_count * 2 * 256;
    const void* kern = big ? (const void*)rts_scatter_kernel<3> : (const void*)rts_scatter_kernel<2>;
    int occ = 0;
    CUDA_TRY(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, 256, 0));
    if (occ < 1) return fail(c, RTS_ECUDA, "rts_scatter_solve_static: kernel does not fit on an SM");
    const int grid = (int)std::max<size_t>(1, std::min<size_t>((size_t)c->sm_count * std::min(occ, 4), (plane_max * nbands + 255) / 256));
    void* args[] = {&p};
    CUDA_TRY(c, cudaLaunchCooperativeKernel(kern, dim3(grid), dim3(256), args, 0, st));
    unsigned long long chg[2 * MAXCHG];
    unsigned flags[4] = {0, 0, 0, 0};
    CUDA_TRY(c, cudaMemcpyAsync(chg, ws + off[5], sizeof(unsigned long long) * nchg, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(c, cudaMemcpyAsync(flags, ws + off[6], sizeof(flags), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(c, cudaStreamSynchronize(st));
    if (flags[1] != 0) return fail(c, RTS_ETIMEOUT, "rts_scatter_solve_static: the grid barrier timed out");
    if (change_host)
        for (size_t q = 0; q < (size_t)niter * nbands; ++q) {                 // [niter][nbands]
            double e, sc;
            std::memcpy(&e, &chg[2 * q], 8); std::memcpy(&sc, &chg[2 * q + 1], 8);
            change_host[q] = (sc > 0.0) ? e / sc : 0.0;
        }
    return RTS_OK;
}

const char* rts_last_error(const rts_ctx* c)
{
    return c ? c->err.c_str() : g_create_err.c_str();
}

}  // extern "C"
