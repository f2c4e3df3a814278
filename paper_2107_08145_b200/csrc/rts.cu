// rts.cu -- host side of the C-ABI in include/rts.h: ray geometry, job list, planner,
// workspace layout, TMA descriptors, launches.  All arithmetic of the path runs in the
// kernels of rts_kernels.cuh; nothing here (or anywhere in the product) touches oracle/.
#include "../../include/rts.h"
#include "rts_kernels.cuh"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
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
    int TV = 0, ntv = 0;
    int userTV = 0;
};

struct HostJob {
    JobDesc d;
    int nsteps;
    int buf;             // exchange-buffer slot
};

}  // namespace

struct rts_ctx {
    int nx = 0, ny = 0, nz = 0, nb = 0;
    double h[3] = {0, 0, 0};
    int npass = 3;
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
    int user_ctas_per_sm = 0;
    // plan
    bool planned = false;
    TypePlan tp[3];
    std::vector<HostJob> jobs;
    int total_tickets = 0, grid = 0, nbuf = 0;
    int ctas_per_sm = 0, threads = 256, smem_bytes = 0;
    int PX = 0, PY = 0;
    size_t ws_bytes = 0;
    // workspace offsets
    size_t off_coefZ = 0, off_coefY = 0, off_coefX = 0, off_QB = 0, off_ksum = 0, off_kstar = 0, off_abort = 0,
           off_jobs = 0, off_prog = 0, off_buf0 = 0, buf_stride = 0, buf_Gu = 0, off_stage_in = 0, off_stage_out = 0;
    size_t prog_ints = 0;
    int nblk_a = 0;
    // workspace
    unsigned char* ws = nullptr;
    size_t ws_have = 0;
    bool maps_ready = false;
    cudaEvent_t ev = nullptr;
    bool timing = false;
    cudaEvent_t tev[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};
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
    r.slot = (r.su < 0) ? 1 : 0;
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
    for (int q = 0; q < 4; ++q) {
        rc.wx[q] = (float)w[q];
        rc.wk[q] = (float)(0.5 * r.ds * w[q]);
    }
    rc.kc = (float)(0.5 * r.ds);
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

int smem_for(int n_u, int TV)
{
    const int n_u4 = (n_u + 3) & ~3;
    const int BOX = (n_u4 + 2 * XPAD) * (TV + 2);
    const int stage = (2 * BOX + 31) & ~31, xf = (NS * BOX + 31) & ~31;
    return (NSTAGE * stage + xf + 2 * NS * (n_u4 + 2 * XPAD)) * (int)sizeof(float);
}
int blocks_for(int n_u, int TV) { return (((n_u + 3) & ~3) >> 2) * ((TV + 1) >> 1); }

// --------------------------------------------------------------------------- planner
// Chooses the band height TV per march axis, builds the job list (ray pairs x bands), the
// ticket order and the exchange-buffer pool.
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
    for (int a = 0; a < 3; ++a) {
        TypePlan& t = c->tp[a];
        t.n_m = n[a];
        t.n_u = (a == 0) ? n[1] : n[0];
        t.n_v = (a == 2) ? n[1] : n[2];
    }
    c->PX = (int)align_up((size_t)c->nx, 4) + 2 * XPAD;
    c->PY = (int)align_up((size_t)c->ny, 4) + 2 * XPAD;

    // --- job skeletons: (march, dir, sv) groups, sub-jobs with <= 1 ray per u-sign slot
    struct Group { int march, dir, sv; std::vector<std::vector<int>> sub; };
    std::vector<Group> groups;
    for (int ri = 0; ri < (int)c->rays.size(); ++ri) {
        const HostRay& r = c->rays[ri];
        Group* g = nullptr;
        for (auto& gg : groups)
            if (gg.march == r.march && gg.dir == r.dir && gg.sv == r.sv) g = &gg;
        if (!g) { groups.push_back(Group{r.march, r.dir, r.sv, {}}); g = &groups.back(); }
        bool placed = false;
        for (auto& sub : g->sub) {
            bool freeslot = true;
            for (int rj : sub) freeslot &= (c->rays[rj].slot != r.slot);
            if (freeslot) { sub.push_back(ri); placed = true; break; }
        }
        if (!placed) g->sub.push_back(std::vector<int>{ri});
    }
    bool used[3] = {false, false, false};
    for (auto& g : groups) used[g.march] = true;

    // --- band height per march axis: one 4x2 block per thread, 2 CTAs per SM if possible
    cudaFuncAttributes fa;
    CUDA_TRY(c, cudaFuncGetAttributes(&fa, rts_sweep_kernel));
    const int threads = 256;
    c->threads = threads;
    int bestR = 0;
    for (int R = (c->user_ctas_per_sm ? c->user_ctas_per_sm : 2); R >= 1 && !bestR; --R) {
        if ((long long)R * threads * fa.numRegs > 65536) continue;
        const int smem_cap = std::min(c->max_smem_optin, (228 * 1024) / R - 1024 - (int)fa.sharedSizeBytes);
        bool ok = true;
        for (int a = 0; a < 3 && ok; ++a) {
            if (!used[a]) { c->tp[a].TV = 2; c->tp[a].ntv = (c->tp[a].n_v + 1) / 2; continue; }
            TypePlan& t = c->tp[a];
            int best = 0;
            for (int TV = 1; TV <= std::min(t.n_v, 32 * MAXC / NS - 2); ++TV) {
                if (t.userTV && TV != t.userTV) continue;
                if (blocks_for(t.n_u, TV) > threads - 32) break;          // the last warp communicates
                if (smem_for(t.n_u, TV) > smem_cap) break;
                if (TV > 1 && (TV & 1) && !t.userTV) continue;      // even heights: full 4x2 blocks
                best = TV;
            }
            if (!best) { ok = false; break; }
            t.TV = best;
            t.ntv = (t.n_v + best - 1) / best;
        }
        if (ok) bestR = R;
        if (c->user_ctas_per_sm) break;
    }
    if (!bestR) return fail(c, RTS_EINVAL, "planner: a row band does not fit (grid too wide: n_u <= 1024, or bad override)");
    c->ctas_per_sm = bestR;
    c->smem_bytes = 0;
    for (int a = 0; a < 3; ++a)
        if (used[a]) c->smem_bytes = std::max(c->smem_bytes, smem_for(c->tp[a].n_u, c->tp[a].TV));
    {
        int occ = 0;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, rts_sweep_kernel, threads, (size_t)c->smem_bytes) != cudaSuccess || occ < 1)
            return fail(c, RTS_ECUDA, "planner: sweep kernel does not fit on an SM");
        c->ctas_per_sm = std::min(bestR, occ);
    }

    // --- materialise jobs in ticket order
    c->jobs.clear();
    int ticket = 0;
    for (auto& g : groups)
        for (auto& sub : g.sub)
            for (int b = 0; b < c->nb; ++b) {
                HostJob hj{};
                JobDesc& d = hj.d;
                std::memset(&d, 0, sizeof d);
                const TypePlan& t = c->tp[g.march];
                d.march = g.march; d.dir = g.dir; d.sv = g.sv; d.band = b;
                d.n_m = t.n_m; d.n_u = t.n_u; d.n_v = t.n_v;
                d.TV = t.TV; d.ntv = t.ntv;
                d.per_v = (g.march == 2) ? 1 : 0;
                d.ticket_begin = ticket;
                ticket += t.ntv;
                d.npass = c->npass;
                d.nz = c->nz;
                const long long nxy = (long long)c->nx * c->ny;
                d.it_sr = nxy; d.it_sb = (long long)c->n_up * nxy;
                const long long PX = c->PX, PY = c->PY;
                // coefficient layouts (one per march axis): rows v contiguous with pitch = box width
                if (g.march == 2)      { d.q_in_B = 0; d.q_sm = nxy;   d.q_sv = c->nx; d.it_su = 1;     d.it_so = c->nx;
                                         d.c_field = (long long)c->nz * (c->ny + 2) * PX; d.c_m = (long long)(c->ny + 2) * PX; d.c_v = PX; d.c_off = PX; }
                else if (g.march == 1) { d.q_in_B = 0; d.q_sm = c->nx; d.q_sv = nxy;   d.it_su = 1;     d.it_so = c->nx;
                                         d.c_field = (long long)c->ny * (c->nz + 2) * PX; d.c_m = (long long)(c->nz + 2) * PX; d.c_v = PX; d.c_off = PX; }
                else                   { d.q_in_B = 1; d.q_sm = c->ny; d.q_sv = nxy;   d.it_su = c->nx; d.it_so = 1;
                                         d.c_field = (long long)c->nx * (c->nz + 2) * PY; d.c_m = (long long)(c->nz + 2) * PY; d.c_v = PY; d.c_off = PY; }
                for (int q = 0; q < NS; ++q) d.ray[q].itop = -1;
                for (int ri : sub) make_ray_consts(c->rays[ri], d.ray[c->rays[ri].slot]);
                hj.nsteps = t.n_m * c->npass;
                c->jobs.push_back(hj);
            }
    c->total_tickets = ticket;
    const int slots = c->sm_count * c->ctas_per_sm;
    c->grid = std::min(slots, c->total_tickets);
    int max_ntv = 1, min_ntv = 1 << 30;
    for (auto& hj : c->jobs) { max_ntv = std::max(max_ntv, hj.d.ntv); min_ntv = std::min(min_ntv, hj.d.ntv); }
    if (max_ntv > c->grid && c->total_tickets > c->grid)
        return fail(c, RTS_EINVAL, "planner: more row bands per job than resident CTAs (grid too tall)");
    // exchange-buffer pool: a slot may be reused once the job that held it must have finished
    c->nbuf = std::min((int)c->jobs.size(), (slots + min_ntv - 1) / min_ntv + 2);
    for (size_t j = 0; j < c->jobs.size(); ++j) c->jobs[j].buf = (int)(j % c->nbuf);

    // --- workspace layout
    const size_t N = (size_t)c->nx * c->ny * c->nz;
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes, 256); return o; };
    const size_t fZ = (size_t)c->nz * (c->ny + 2) * c->PX;
    const size_t fY = (size_t)c->ny * (c->nz + 2) * c->PX;
    const size_t fX = (size_t)c->nx * (c->nz + 2) * c->PY;
    c->off_coefZ = take(sizeof(float) * fZ * 2 * c->nb);
    c->off_coefY = take(sizeof(float) * fY * 2 * c->nb);
    c->off_coefX = take(sizeof(float) * fX * 2 * c->nb);
    c->off_QB = take(sizeof(float) * N);
    c->nblk_a = ((c->nx + 31) / 32) * ((c->ny + 31) / 32);
    c->off_ksum = take(sizeof(double) * (size_t)c->nb * c->nz * c->nblk_a);
    c->off_kstar = take(sizeof(int) * c->nb);
    c->off_abort = take(sizeof(int) * 8);                    // [0] watchdog, [1] ticket counter
    c->off_jobs = take(sizeof(JobDesc) * c->jobs.size());
    c->prog_ints = (size_t)c->total_tickets;
    c->off_prog = take(sizeof(int) * c->prog_ints);
    size_t mH = 0, mG = 0;
    for (auto& hj : c->jobs) {
        const JobDesc& d = hj.d;
        const size_t n_u4 = (size_t)((d.n_u + 3) & ~3);
        mH = std::max(mH, (size_t)d.ntv * hj.nsteps * NS * n_u4);
        mG = std::max(mG, (size_t)d.ntv * 2 * d.n_m * NS * d.TV);
    }
    c->buf_Gu = align_up(sizeof(float) * mH, 256);
    c->buf_stride = c->buf_Gu + align_up(sizeof(float) * mG, 256);
    c->off_buf0 = take(c->buf_stride * c->nbuf);
    c->off_stage_in = take(sizeof(float) * N * 3);
    c->off_stage_out = take(sizeof(float) * (N + (size_t)c->nb * c->n_up * c->ny * c->nx));
    c->ws_bytes = off;
    c->planned = true;
    return RTS_OK;
}

int bind_workspace(rts_ctx* c)
{
    unsigned char* ws = c->ws;
    float* coefL[3] = {(float*)(ws + c->off_coefX), (float*)(ws + c->off_coefY), (float*)(ws + c->off_coefZ)};
    std::vector<JobDesc> flat;
    for (auto& hj : c->jobs) {
        JobDesc& d = hj.d;
        unsigned char* sb = ws + c->off_buf0 + c->buf_stride * hj.buf;
        d.Hrow = (float*)sb;
        d.Gu = (float*)(sb + c->buf_Gu);
        d.progress = (int*)(ws + c->off_prog) + d.ticket_begin;
        d.kstar = (const int*)(ws + c->off_kstar) + d.band;
        d.cbase = coefL[d.march] + (size_t)(2 * d.band) * d.c_field;
        flat.push_back(d);
    }
    CUDA_TRY(c, cudaMemcpy(ws + c->off_jobs, flat.data(), sizeof(JobDesc) * flat.size(), cudaMemcpyHostToDevice));
    CUDA_TRY(c, cudaMemset(ws + c->off_abort, 0, sizeof(int) * 8));   // status word: a fresh workspace holds garbage
    c->maps_ready = true;
    return RTS_OK;
}

cudaStream_t as_stream(void* s) { return (cudaStream_t)s; }

int launch_stage_a(rts_ctx* c, const float* rho, const float* T, const float* P, float* plain_k, float* plain_s,
                   cudaStream_t st)
{
    CoefParams p{};
    p.nx = c->nx; p.ny = c->ny; p.nz = c->nz; p.nb = c->nb; p.nT = c->nT; p.nP = c->nP;
    p.logT_min = c->logT_min; p.inv_dT = (c->nT - 1) / (c->logT_max - c->logT_min);
    p.logP_min = c->logP_min; p.inv_dP = (c->nP - 1) / (c->logP_max - c->logP_min);
    p.logkappa = c->d_logkappa; p.bandfrac = c->d_bandfrac;
    p.rho = rho; p.T = T; p.P = P;
    p.coefZ = (float*)(c->ws + c->off_coefZ); p.coefY = (float*)(c->ws + c->off_coefY); p.coefX = (float*)(c->ws + c->off_coefX);
    p.PX = c->PX; p.PY = c->PY;
    p.strideZ_f = (long long)c->nz * (c->ny + 2) * c->PX;
    p.strideY_f = (long long)c->ny * (c->nz + 2) * c->PX;
    p.strideX_f = (long long)c->nx * (c->nz + 2) * c->PY;
    p.ksum = (double*)(c->ws + c->off_ksum);
    p.plain_k = plain_k; p.plain_s = plain_s;
    dim3 grid((c->nx + 31) / 32, (c->ny + 31) / 32, c->nz), block(32, 8);
    rts_coef_kernel<<<grid, block, 0, st>>>(p);
    CUDA_TRY(c, cudaGetLastError());
    return RTS_OK;
}

}  // namespace

// =========================================================================== C-ABI
extern "C" {

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
    if ((e = cudaFuncGetAttributes(&fa, rts_sweep_kernel)) != cudaSuccess) return bail(std::string("sweep kernel not loadable: ") + cudaGetErrorString(e));
    c->max_smem_optin = (int)prop.sharedMemPerBlockOptin - (int)fa.sharedSizeBytes;
    if ((e = cudaFuncSetAttribute(rts_sweep_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, c->max_smem_optin)) != cudaSuccess)
        return bail(std::string("cudaFuncSetAttribute(max dynamic smem): ") + cudaGetErrorString(e));
    if ((e = cudaEventCreateWithFlags(&c->ev, cudaEventDisableTiming)) != cudaSuccess) return bail(cudaGetErrorString(e));
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
    (void)tile_u;   // tiles always span the full unit-stride extent
    if (march < 0 || march > 2 || tile_v < 0 || tile_v > 32 * MAXC / NS - 2)
        return fail(c, RTS_EINVAL, "rts_set_tiling: bad argument");
    c->tp[march].userTV = tile_v;
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
    int v[12] = {4, c->total_tickets, c->ctas_per_sm, (int)c->jobs.size(), c->threads, c->smem_bytes,
                 c->grid, c->nbuf, c->tp[0].TV, c->tp[1].TV, c->tp[2].TV, 0};
    for (int i = 0; i < n && i < 12; ++i) what[i] = v[i];
    return RTS_OK;
}

int rts_coefficients(rts_ctx* c, const float* rho, const float* T, const float* P, float* kaprho, float* S, void* stream)
{
    if (!c) return RTS_EINVAL;
    if (!rho || !T || !P || !kaprho || !S) return fail(c, RTS_EINVAL, "rts_coefficients: null pointer");
    if (!c->have_tables || !c->ws || !c->planned || !c->maps_ready) return fail(c, RTS_ESTATE, "rts_coefficients: tables/workspace not set");
    return launch_stage_a(c, rho, T, P, kaprho, S, as_stream(stream));
}

int rts_solve(rts_ctx* c, const float* rho, const float* T, const float* P, float* Q, float* Itop, void* stream)
{
    if (!c) return RTS_EINVAL;
    if (!rho || !T || !P || !Q) return fail(c, RTS_EINVAL, "rts_solve: null pointer");
    if (!c->have_tables) return fail(c, RTS_ESTATE, "rts_solve: tables not set");
    if (!c->ws || !c->planned || !c->maps_ready) return fail(c, RTS_ESTATE, "rts_solve: workspace not set (or configuration changed since)");
    cudaStream_t st = as_stream(stream);
    const size_t N = (size_t)c->nx * c->ny * c->nz;
    unsigned char* ws = c->ws;

    // stage A + switch heights
    if (c->timing) CUDA_TRY(c, cudaEventRecord(c->tev[0], st));
    int rc = launch_stage_a(c, rho, T, P, nullptr, nullptr, st);
    if (rc != RTS_OK) return rc;
    rts_kstar_kernel<<<1, 32, 0, st>>>((const double*)(ws + c->off_ksum), c->nb, c->nz, c->nblk_a,
                                       1.0 / ((double)c->nx * c->ny), c->h[2], 5.0, (int*)(ws + c->off_kstar));
    CUDA_TRY(c, cudaGetLastError());
    if (c->timing) CUDA_TRY(c, cudaEventRecord(c->tev[1], st));

    // outputs start from zero; x-march sweeps accumulate into the y-fastest QB
    float* QB = (float*)(ws + c->off_QB);
    CUDA_TRY(c, cudaMemsetAsync(Q, 0, N * sizeof(float), st));
    CUDA_TRY(c, cudaMemsetAsync(QB, 0, N * sizeof(float), st));
    CUDA_TRY(c, cudaMemsetAsync(ws + c->off_abort, 0, sizeof(int) * 8, st));

    CUDA_TRY(c, cudaMemsetAsync(ws + c->off_prog, 0, sizeof(int) * c->prog_ints, st));
    // the sweep: one persistent launch, tasks handed out by an in-order ticket counter
    if (c->timing) CUDA_TRY(c, cudaEventRecord(c->tev[2], st));
    {
        const JobDesc* djobs = (const JobDesc*)(ws + c->off_jobs);
        int* abortf = (int*)(ws + c->off_abort);
        rts_sweep_kernel<<<c->grid, c->threads, (size_t)c->smem_bytes, st>>>(
            djobs, (int)c->jobs.size(), c->total_tickets, abortf + 1, Q, QB, Itop, abortf);
        CUDA_TRY(c, cudaGetLastError());
    }
    // finalize
    if (c->timing) CUDA_TRY(c, cudaEventRecord(c->tev[3], st));
    {
        dim3 grid((c->nx + 31) / 32, (c->ny + 31) / 32, c->nz), block(32, 8);
        rts_finalize_kernel<<<grid, block, 0, st>>>(Q, QB, c->nx, c->ny, c->nz);
        CUDA_TRY(c, cudaGetLastError());
    }
    if (c->timing) CUDA_TRY(c, cudaEventRecord(c->tev[4], st));
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
        int ab = 0;
        e = cudaMemcpy(&ab, c->ws + c->off_abort, sizeof(int), cudaMemcpyDeviceToHost);
        if (e != cudaSuccess) return fail(c, RTS_ECUDA, std::string("status read: ") + cudaGetErrorString(e));
        if (ab) {
            char buf[128];
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
    CUDA_TRY(c, cudaMemcpyAsync(din, rho, N * sizeof(float), cudaMemcpyHostToDevice, st));
    CUDA_TRY(c, cudaMemcpyAsync(din + N, T, N * sizeof(float), cudaMemcpyHostToDevice, st));
    CUDA_TRY(c, cudaMemcpyAsync(din + 2 * N, P, N * sizeof(float), cudaMemcpyHostToDevice, st));
    int rc = rts_solve(c, din, din + N, din + 2 * N, dout, Itop ? dout + N : nullptr, stream);
    if (rc != RTS_OK) return rc;
    CUDA_TRY(c, cudaMemcpyAsync(Q, dout, N * sizeof(float), cudaMemcpyDeviceToHost, st));
    if (Itop) CUDA_TRY(c, cudaMemcpyAsync(Itop, dout + N, nI * sizeof(float), cudaMemcpyDeviceToHost, st));
    return rts_sync_check(c, stream);
}

#ifdef RTS_TRACE
int rts_debug_trace(unsigned long long* out, int n)
{
    return cudaMemcpyFromSymbol(out, rts::g_trace, sizeof(unsigned long long) * n) == cudaSuccess ? 0 : -3;
}
#endif

const char* rts_last_error(const rts_ctx* c)
{
    return c ? c->err.c_str() : g_create_err.c_str();
}

}  // extern "C"
