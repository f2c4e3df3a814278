// rts_kernels.cuh -- device code of the RTS hot path (sm_100a).
//
//   K_a  rts_coef_kernel    stage A  (paper's interpol())
//   K_k  rts_kstar_kernel   picks, per band, the height below which the sweep carries the
//                           departure I - S instead of I (precision device)
//   K_b  rts_sweep_kernel   stages B-E (paper's integrate() + readbuf/writebuf/exchange with
//                           the box as its own neighbour + flux())
//   K_f  rts_finalize_kernel adds the x-march partial heating (stored y-fastest) into Q_rad
//
// Shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <cuda.h>
#include <stdint.h>

namespace rts {

constexpr int   NSLOT = 4;          // rays per sweep job: one per sign pattern (su, sv)
constexpr int   XPAD = 4;           // ghost columns on each side of the unit-stride axis
constexpr float LOG2E = 1.4426950408889634f;
constexpr float FOUR_PI = 12.566370614359172f;
constexpr float DTAU_SERIES = 0.05f; // below this the psi weights come from their series
constexpr double SIGMA_SB_D = 5.670374e-5;
constexpr double PI_D = 3.14159265358979323846;

struct alignas(16) RayC {
    float wx[4];      // bilinear weights of (u,v) (u-su,v) (u,v-sv) (u-su,v-sv); sum == 1 exactly
    float wk[4];      // 0.5*ds*wx  (opacity -> optical path)
    float kc;         // 0.5*ds
    float wq;         // quadrature weight (0: empty slot)
    int   active;
    int   up;         // mu_z > 0
    int   dir_row;    // x/y-march: Dirichlet row in v (0 or nz-1); z-march: unused
    int   itop;       // index among the upward rays, or -1
    int   pad0, pad1;
};

struct JobDesc {
    int march;        // 0: x, 1: y, 2: z  (axis the sweep marches along)
    int dir;          // +1 / -1
    int band;
    int n_m, n_u, n_v;
    int TU, TV, ntu, ntv;
    int per_v;        // v periodic (z-march: v = y) or bounded (x/y-march: v = z)
    int cta_begin, ntiles;
    int npass;
    int nz;
    int q_in_B;       // heating goes to the y-fastest partial buffer (x-march)
    RayC ray[NSLOT];
    float* Dg;        // [2][NSLOT][n_v][n_u]   tile-edge exchange, indexed by step parity
    float* Gu;        // [2][NSLOT][n_m][n_v]   far-u face history, indexed by pass parity
    float* Gv;        // [2][NSLOT][n_m][n_u]   far-v face history (per_v only)
    int*   progress;  // [ntiles] completed steps
    long long q_sm, q_sv;                 // heating strides along (march, v); u stride 1
    long long it_su, it_so, it_sr, it_sb; // I_top strides along u, other axis, ray, band
    const int* kstar; // device: per band switch height
};

// --------------------------------------------------------------------------- PTX helpers
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity) {
    uint32_t ok;
    asm volatile("{\n\t.reg .pred p;\n\t"
                 "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
                 "selp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    return ok != 0;
}
__device__ __forceinline__ void tma_load_4d(void* dst, const CUtensorMap* map, uint64_t* bar,
                                            int c0, int c1, int c2, int c3) {
    asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes"
                 " [%0], [%1, {%3, %4, %5, %6}], [%2];"
                 ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
                 : "memory");
}
__device__ __forceinline__ int ld_acquire(const int* p) {
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release(int* p, int v) {
    asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ float ex2_approx(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float rcp_approx(float x) {
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// =========================================================================== K_a
// Stage A.  One thread block = a 32x32 (x,y) patch of one z level; 32x8 threads, 4 nodes each.
// Evaluates the table coordinates, 10^x and T^4 in fp64 and rounds once to fp32 (DESIGN.md,
// "precision").  Writes kaprho_b, S_b
//   layout A  coefA[b][f][nz][ny+2][PX]   x fastest, x index offset XPAD, y offset 1, periodic
//                                          ghost columns / rows filled here
//   layout B  coefB[b][f][nz][nx][PY]     y fastest, y index offset XPAD, periodic ghosts in y
// and per-block partial sums of kaprho for K_k.
struct CoefParams {
    int nx, ny, nz, nb, nT, nP;
    double logT_min, inv_dT, logP_min, inv_dP;   // inv_d = (n-1)/(max-min)
    const float* logkappa;   // device [nb][nT][nP]
    const float* bandfrac;   // device [nb][nT]
    const float *rho, *T, *P;
    float* coefA; int PX; long long strideA_f;   // field stride = nz*(ny+2)*PX
    float* coefB; int PY; long long strideB_f;   // field stride = nz*nx*PY
    double* ksum;            // [nb][nz][nblk] partial sums (nblk = gridDim.x*gridDim.y), or null
    float* plain_k; float* plain_s;              // optional [nb][N] outputs (rts_coefficients)
};

__global__ void __launch_bounds__(256) rts_coef_kernel(const CoefParams p)
{
    __shared__ float tile[2][32][33];
    __shared__ double red[8];
    const int tx = threadIdx.x, ty = threadIdx.y;
    const int i0 = blockIdx.x * 32, j0 = blockIdx.y * 32, k = blockIdx.z;
    const int i = i0 + tx;
    const long long N = (long long)p.nx * p.ny * p.nz;

    // band-independent part, 4 nodes per thread (rows ty, ty+8, ty+16, ty+24)
    double t_[4], u_[4], planck[4], rho_[4];
    int it_[4], ip_[4];
    bool ok[4];
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        const int j = j0 + ty + 8 * r;
        ok[r] = (i < p.nx) && (j < p.ny);
        t_[r] = u_[r] = planck[r] = rho_[r] = 0.0;
        it_[r] = ip_[r] = 0;
        if (ok[r]) {
            const long long n = ((long long)k * p.ny + j) * p.nx + i;
            const double Tn = (double)p.T[n], Pn = (double)p.P[n];
            double xT = (log10(Tn) - p.logT_min) * p.inv_dT;
            double xP = (log10(Pn) - p.logP_min) * p.inv_dP;
            xT = fmin(fmax(xT, 0.0), (double)(p.nT - 1));
            xP = fmin(fmax(xP, 0.0), (double)(p.nP - 1));
            int a = (int)floor(xT); if (a > p.nT - 2) a = p.nT - 2;
            int b = (int)floor(xP); if (b > p.nP - 2) b = p.nP - 2;
            it_[r] = a; ip_[r] = b;
            t_[r] = xT - a; u_[r] = xP - b;
            planck[r] = SIGMA_SB_D * (Tn * Tn) * (Tn * Tn) / PI_D;
            rho_[r] = (double)p.rho[n];
        }
    }

    for (int b = 0; b < p.nb; ++b) {
        const float* L = p.logkappa + (size_t)b * p.nT * p.nP;
        const float* F = p.bandfrac + (size_t)b * p.nT;
        float* A0 = p.coefA + (size_t)(2 * b) * p.strideA_f;
        float* A1 = A0 + p.strideA_f;
        double part = 0.0;
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            float kr = 0.f, sr = 0.f;
            if (ok[r]) {
                const int a = it_[r], c = ip_[r];
                const double t = t_[r], u = u_[r];
                const double l00 = (double)L[(size_t)a * p.nP + c], l10 = (double)L[(size_t)(a + 1) * p.nP + c];
                const double l01 = (double)L[(size_t)a * p.nP + c + 1], l11 = (double)L[(size_t)(a + 1) * p.nP + c + 1];
                const double lk = (1.0 - t) * (1.0 - u) * l00 + t * (1.0 - u) * l10 + (1.0 - t) * u * l01 + t * u * l11;
                const double fb = (1.0 - t) * (double)F[a] + t * (double)F[a + 1];
                const double kd = exp10(lk) * rho_[r];
                kr = (float)kd;
                sr = (float)(fb * planck[r]);
                part += kd;
                const int j = j0 + ty + 8 * r;
                // layout A with periodic images
                const int jrows[3] = {j + 1, (j == 0) ? p.ny + 1 : -1, (j == p.ny - 1) ? 0 : -1};
                const int icols[3] = {i + XPAD, (i < XPAD && i + p.nx + XPAD < p.PX) ? i + p.nx + XPAD : -1,
                                      (i >= p.nx - XPAD && i - p.nx + XPAD >= 0) ? i - p.nx + XPAD : -1};
#pragma unroll
                for (int a2 = 0; a2 < 3; ++a2) {
                    if (jrows[a2] < 0) continue;
                    const size_t rowoff = ((size_t)k * (p.ny + 2) + jrows[a2]) * p.PX;
#pragma unroll
                    for (int c2 = 0; c2 < 3; ++c2) {
                        if (icols[c2] < 0) continue;
                        A0[rowoff + icols[c2]] = kr;
                        A1[rowoff + icols[c2]] = sr;
                    }
                }
                if (p.plain_k) {
                    const long long n = ((long long)k * p.ny + j) * p.nx + i;
                    p.plain_k[(size_t)b * N + n] = kr;
                    p.plain_s[(size_t)b * N + n] = sr;
                }
            }
            tile[0][ty + 8 * r][tx] = kr;
            tile[1][ty + 8 * r][tx] = sr;
        }
        // block sum of kaprho (deterministic order)
        if (p.ksum) {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
            if (tx == 0) red[ty] = part;
        }
        __syncthreads();
        if (p.ksum && tx == 0 && ty == 0) {
            double s = 0.0;
            for (int w = 0; w < 8; ++w) s += red[w];
            const int nblk = gridDim.x * gridDim.y;
            p.ksum[((size_t)b * p.nz + k) * nblk + blockIdx.y * gridDim.x + blockIdx.x] = s;
        }
        // layout B: transposed write, coalesced along y
        float* B0 = p.coefB + (size_t)(2 * b) * p.strideB_f;
        float* B1 = B0 + p.strideB_f;
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const int ii = i0 + ty + 8 * r, jj = j0 + tx;
            if (ii < p.nx && jj < p.ny) {
                const float kr = tile[0][tx][ty + 8 * r], sr = tile[1][tx][ty + 8 * r];
                const size_t rowoff = ((size_t)k * p.nx + ii) * p.PY;
                const int jc[3] = {jj + XPAD, (jj < XPAD && jj + p.ny + XPAD < p.PY) ? jj + p.ny + XPAD : -1,
                                   (jj >= p.ny - XPAD && jj - p.ny + XPAD >= 0) ? jj - p.ny + XPAD : -1};
#pragma unroll
                for (int c2 = 0; c2 < 3; ++c2) {
                    if (jc[c2] < 0) continue;
                    B0[rowoff + jc[c2]] = kr;
                    B1[rowoff + jc[c2]] = sr;
                }
            }
        }
        __syncthreads();
    }
}

// =========================================================================== K_k
// kstar[b] = highest level k whose horizontally averaged optical depth from the top,
// tau(k) = sum_{k' >= k} <kaprho_b>(k') dz, is >= tau_switch; -1 if none.  One block.
__global__ void rts_kstar_kernel(const double* ksum, int nb, int nz, int nblk, double inv_nxy,
                                 double dz, double tau_switch, int* kstar)
{
    for (int b = threadIdx.x; b < nb; b += blockDim.x) {
        double tau = 0.0;
        int ks = -1;
        for (int k = nz - 1; k >= 0; --k) {
            double s = 0.0;
            const double* q = ksum + ((size_t)b * nz + k) * nblk;
            for (int w = 0; w < nblk; ++w) s += q[w];
            tau += s * inv_nxy * dz;
            if (tau >= tau_switch) { ks = k; break; }
        }
        kstar[b] = ks;
    }
}

// =========================================================================== K_b
// Persistent lockstep sweep.  One CTA = one tile (TU x TV nodes of the march plane) of one
// job (march axis+direction, band, up to 4 rays = the 4 transverse sign patterns).  The CTA
// marches plane by plane through all passes; per step it
//   1. waits until its (up to 8, periodic) neighbour tiles have finished the previous step,
//   2. fills the one-node ring of its carried-quantity planes from the neighbours' published
//      edge values (same pass) or from the far-face history of the previous pass (periodic
//      seam: Jacobi ghosts),
//   3. updates all nodes x rays (opacity / source planes staged by TMA, double buffered),
//   4. publishes its edge values and its step counter (release).
// Carried quantity: X = I - a*S with a = 1 at levels k <= kstar (optically thick part, where
// J - S would cancel) and a = 0 above (thin part, where I << S would cancel).
struct SweepSmem {
    float* coef[2];   // [stage] -> [2 fields][BOXV][BOXU]
    float* X[2];      // [buffer] -> [NSLOT][BOXV][BOXU]
};

template <int SU, int SV>
__device__ __forceinline__ void ray_quad_update(
    const float (&kf)[3][6], const float (&sf)[3][6], const float (&kp)[4], const float (&sp)[4],
    const float* __restrict__ Xold, int base, int BOXU, const RayC& rc,
    const float ap, const float a0, const float a1, float (&xp)[4])
{
    // own row and upwind row of the carried quantity
    const int rowu = base - SV * BOXU;
    const float4 x0 = *reinterpret_cast<const float4*>(Xold + base);
    const float4 x1 = *reinterpret_cast<const float4*>(Xold + rowu);
    const float e0 = Xold[base + (SU > 0 ? -1 : 4)];
    const float e1 = Xold[rowu + (SU > 0 ? -1 : 4)];
    const float xo[4] = {x0.x, x0.y, x0.z, x0.w};
    const float xu[4] = {x1.x, x1.y, x1.z, x1.w};
    float xos[4], xus[4];
    if (SU > 0) { xos[0] = e0; xos[1] = xo[0]; xos[2] = xo[1]; xos[3] = xo[2];
                  xus[0] = e1; xus[1] = xu[0]; xus[2] = xu[1]; xus[3] = xu[2]; }
    else        { xos[0] = xo[1]; xos[1] = xo[2]; xos[2] = xo[3]; xos[3] = e0;
                  xus[0] = xu[1]; xus[1] = xu[2]; xus[2] = xu[3]; xus[3] = e1; }
    constexpr int RU = 1 - SV;   // row index of the upwind row in kf/sf
    const float w0 = rc.wx[0], w1 = rc.wx[1], w2 = rc.wx[2], w3 = rc.wx[3];
    const float k0 = rc.wk[0], k1 = rc.wk[1], k2 = rc.wk[2], k3 = rc.wk[3], kc = rc.kc;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const int c = j + 1, cs = j + 1 - SU;
        const float Xu = w0 * xo[j] + w1 * xos[j] + w2 * xu[j] + w3 * xus[j];
        const float dt = kc * kp[j] + k0 * kf[1][c] + k1 * kf[1][cs] + k2 * kf[RU][c] + k3 * kf[RU][cs];
        const float R0 = w0 * sf[1][c] + w1 * sf[1][cs];
        const float R1 = w2 * sf[RU][c] + w3 * sf[RU][cs];
        const float St = a0 * R0 + a1 * R1;        // departure-carried part of S_u
        const float Sh = (R0 + R1) - St;           // directly integrated part of S_u
        const float Stp = ap * sp[j];
        const float Shp = sp[j] - Stp;
        const float dS = Stp - St;
        // psi weights: closed form, or series below DTAU_SERIES
        const float E = ex2_approx(-dt * LOG2E);
        const float omE = 1.0f - E;
        const float w1b = omE * rcp_approx(dt);
        const float pps = dt * (0.5f - dt * (1.0f / 6.0f - dt * (1.0f / 24.0f - dt * (1.0f / 120.0f))));
        const float pus = dt * (0.5f - dt * (1.0f / 3.0f - dt * (1.0f / 8.0f - dt * (1.0f / 30.0f))));
        const bool sm = dt < DTAU_SERIES;
        const float wl = sm ? 1.0f - pps : w1b;     // (1-E)/dtau
        const float pp = sm ? pps : 1.0f - w1b;     // psi_p
        const float pu = sm ? pus : w1b - E;        // psi_u
        const float em1 = sm ? dt * wl : omE;       // 1 - E
        float v = fmaf(-Xu, em1, Xu);
        v = fmaf(-dS, wl, v);
        v = fmaf(pu, Sh, v);
        v = fmaf(pp, Shp, v);
        xp[j] = v;
    }
}

__device__ __forceinline__ bool spin_abort(const int* abortf, unsigned& spins)
{
    if ((++spins & 1023u) == 0u) {
        if (*reinterpret_cast<const volatile int*>(abortf) != 0) return true;
        if (spins > (1u << 26)) { atomicExch(const_cast<int*>(abortf), 1); return true; }
    }
    return false;
}

__global__ void __launch_bounds__(256, 2)
rts_sweep_kernel(const __grid_constant__ CUtensorMap mapX, const __grid_constant__ CUtensorMap mapY,
                 const __grid_constant__ CUtensorMap mapZ, const JobDesc* __restrict__ jobs, int njobs,
                 float* __restrict__ Qa, float* __restrict__ Qb, float* __restrict__ Itop_all, int* abortf)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ JobDesc J;
    __shared__ __align__(8) uint64_t mbar[2];
    __shared__ int s_nbr[8];
    __shared__ int s_nnbr;
    __shared__ int s_abort;

    // ---- locate job / tile
    {
        int jid = 0;
        for (int q = 1; q < njobs; ++q)
            if ((int)blockIdx.x >= jobs[q].cta_begin) jid = q;
        const int* src = reinterpret_cast<const int*>(jobs + jid);
        int* dst = reinterpret_cast<int*>(&J);
        for (int w = threadIdx.x; w < (int)(sizeof(JobDesc) / sizeof(int)); w += blockDim.x) dst[w] = src[w];
    }
    __syncthreads();
    const int tile = (int)blockIdx.x - J.cta_begin;
    if (tile >= J.ntiles) return;
    const int ta = tile % J.ntu, tb = tile / J.ntu;
    const int TU = J.TU, TV = J.TV;
    const int BOXU = TU + 2 * XPAD, BOXV = TV + 2;
    const int BOX = BOXU * BOXV;
    const int u0 = ta * TU, v0 = tb * TV;
    const int tu = min(TU, J.n_u - u0), tv = min(TV, J.n_v - v0);
    const int n_u = J.n_u, n_v = J.n_v, n_m = J.n_m;
    const bool zmarch = (J.march == 2);
    const int nsteps = n_m * J.npass;
    const int kstar = *J.kstar;
    const CUtensorMap* map = (J.march == 0) ? &mapX : (J.march == 1) ? &mapY : &mapZ;
    float* const Qdst = J.q_in_B ? Qb : Qa;
    float* const Itop_b = Itop_all ? Itop_all + (long long)J.band * J.it_sb : nullptr;

    // ---- shared memory carve-up
    const int stage_floats = (2 * BOX + 31) & ~31;
    const int xbuf_floats = (NSLOT * BOX + 31) & ~31;
    float* sm_f = reinterpret_cast<float*>(smem_raw);
    SweepSmem S;
    S.coef[0] = sm_f;
    S.coef[1] = sm_f + stage_floats;
    S.X[0] = sm_f + 2 * stage_floats;
    S.X[1] = S.X[0] + xbuf_floats;
    const uint32_t stage_bytes = (uint32_t)(2 * BOX * sizeof(float));

    // ---- neighbour list (torus in u; in v only if periodic)
    if (threadIdx.x == 0) {
        int n = 0;
        for (int db = -1; db <= 1; ++db)
            for (int da = -1; da <= 1; ++da) {
                if (da == 0 && db == 0) continue;
                int a = ta + da, b = tb + db;
                if (a < 0) a += J.ntu; else if (a >= J.ntu) a -= J.ntu;
                if (b < 0 || b >= J.ntv) {
                    if (!J.per_v) continue;
                    if (b < 0) b += J.ntv; else b -= J.ntv;
                }
                const int t2 = b * J.ntu + a;
                if (t2 == tile) continue;
                bool dup = false;
                for (int q = 0; q < n; ++q) dup |= (s_nbr[q] == t2);
                if (!dup) s_nbr[n++] = t2;
            }
        s_nnbr = n;
        s_abort = 0;
        mbar_init(&mbar[0], 1);
        mbar_init(&mbar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    // TMA coordinates of the box of march plane `pl`
    auto issue_load = [&](int L) {
        // L = load number (-1: the plane "before" step 0), stage = L & 1
        int m = (L < 0) ? n_m - 1 : (L % n_m);
        const int pl = (J.dir > 0) ? m : n_m - 1 - m;
        const int st = L & 1;
        uint64_t* bar = &mbar[st];
        mbar_expect_tx(bar, stage_bytes);
        if (J.march == 2)      tma_load_4d(S.coef[st], map, bar, u0, v0, pl, 2 * J.band);        // (x, y+1-1, z)
        else if (J.march == 1) tma_load_4d(S.coef[st], map, bar, u0, pl + 1, v0 - 1, 2 * J.band); // (x, y, z)
        else                   tma_load_4d(S.coef[st], map, bar, u0, pl, v0 - 1, 2 * J.band);     // (y, x, z)
    };
    if (threadIdx.x == 0) {
        issue_load(-1);
        issue_load(0);
    }

    const int quads_u = (tu + 3) >> 2;
    const int nquads = quads_u * tv;
    int* const my_progress = J.progress + tile;
    const size_t plane_uv = (size_t)n_v * n_u;
    const bool last_possible = true;
    (void)last_possible;

    for (int s = 0; s < nsteps; ++s) {
        const int m = s % n_m;
        const int pass = s / n_m;
        const int pl = (J.dir > 0) ? m : n_m - 1 - m;
        const int plprev = pl - J.dir;                 // plane of the previous step (may be out of range at m == 0)
        const int mprev = (m == 0) ? n_m - 1 : m - 1;
        const int st = s & 1;
        const float* Bc = S.coef[st];                  // plane of this step (centres)
        const float* Bp = S.coef[st ^ 1];              // previous plane (upwind neighbourhood)
        float* Xold = S.X[s & 1];
        float* Xnew = S.X[(s & 1) ^ 1];
        const bool lastpass = (pass == J.npass - 1);

        // ---- 1. wait for neighbours (warp 0) and for the TMA of this step's plane
        if (s > 0 && threadIdx.x < 32) {
            const int nn = s_nnbr;
            unsigned spins = 0;
            bool ok = false;
            while (!ok) {
                int v = s;
                if ((int)threadIdx.x < nn) v = ld_acquire(J.progress + s_nbr[threadIdx.x]);
                ok = __all_sync(0xffffffffu, v >= s);
                if (!ok) {
                    bool ab = spin_abort(abortf, spins);
                    if (__any_sync(0xffffffffu, ab)) { if (threadIdx.x == 0) s_abort = 1; break; }
                    __nanosleep(64);
                }
            }
        }
        {
            unsigned spins = 0;
            const uint32_t par = (uint32_t)(((s + 1) >> 1) & 1);
            while (!mbar_try_wait(&mbar[st], par)) { if (spin_abort(abortf, spins)) { s_abort = 1; break; } }
            if (s == 0) {
                spins = 0;
                while (!mbar_try_wait(&mbar[1], 0u)) { if (spin_abort(abortf, spins)) { s_abort = 1; break; } }
            }
        }
        __syncthreads();
        if (s_abort) return;

        const bool dirichlet_plane = zmarch && (m == 0);
        const float a_pl = (pl <= kstar) ? 1.f : 0.f;          // z-march: a of this plane
        const float a_plprev = (plprev <= kstar) ? 1.f : 0.f;  // z-march: a of the previous plane

        // ---- 2. ring (and, at the very first step, the whole plane) of the carried quantity
        if (!dirichlet_plane) {
            const float* Sp_prev = Bp + BOX;   // source function of the previous plane
            if (s == 0) {
                // X^(0) = I^(0) - a S on the plane "before" step 0 (x/y-march only reach here)
                for (int idx = threadIdx.x; idx < NSLOT * BOX; idx += blockDim.x) {
                    const int q = idx / BOX, pos = idx - q * BOX;
                    const int vl = pos / BOXU - 1;
                    const int gv = v0 + vl;
                    const float Sv = Sp_prev[pos];
                    const float a = (gv <= kstar) ? 1.f : 0.f;
                    const bool dnode = (gv == J.ray[q].dir_row);
                    const float I0 = (dnode && !J.ray[q].up) ? 0.f : Sv;
                    Xold[idx] = I0 - a * Sv;
                }
            } else {
                const int ncol = tv + 2;                 // ring column: vl = -1 .. tv
                const int per_slot = ncol + tu;          // + ring row: ul = 0 .. tu-1
                for (int idx = threadIdx.x; idx < NSLOT * per_slot; idx += blockDim.x) {
                    const int q = idx / per_slot, e = idx - q * per_slot;
                    const RayC& rc = J.ray[q];
                    if (!rc.active) continue;
                    const int su = (q & 1) ? -1 : 1, sv = (q & 2) ? -1 : 1;
                    int ul, vl;
                    if (e < ncol) { ul = (su > 0) ? -1 : tu; vl = e - 1; }
                    else          { ul = e - ncol; vl = (sv > 0) ? -1 : tv; }
                    const int pos = (vl + 1) * BOXU + ul + XPAD;
                    int gu = u0 + ul, gv = v0 + vl;
                    float val = 0.f;
                    bool wrapped = false;
                    if (gu < 0) { gu += n_u; wrapped = true; } else if (gu >= n_u) { gu -= n_u; wrapped = true; }
                    bool outside = false;
                    if (gv < 0 || gv >= n_v) {
                        if (J.per_v) { gv += (gv < 0) ? n_v : -n_v; wrapped = true; }
                        else outside = true;
                    }
                    if (!outside) {
                        if (wrapped) {
                            if (pass == 0) {
                                const float Sv = Sp_prev[pos];
                                const float a = zmarch ? a_plprev : ((gv <= kstar) ? 1.f : 0.f);
                                const bool dnode = zmarch ? (mprev == 0) : (gv == rc.dir_row);
                                const float I0 = (dnode && !rc.up) ? 0.f : Sv;
                                val = I0 - a * Sv;
                            } else {
                                const int pb = (pass - 1) & 1;
                                const bool wu = (u0 + ul < 0) || (u0 + ul >= n_u);
                                if (wu) val = __ldcg(J.Gu + (((size_t)pb * NSLOT + q) * n_m + mprev) * n_v + gv);
                                else    val = __ldcg(J.Gv + (((size_t)pb * NSLOT + q) * n_m + mprev) * n_u + gu);
                            }
                        } else {
                            val = __ldcg(J.Dg + ((size_t)((s - 1) & 1) * NSLOT + q) * plane_uv + (size_t)gv * n_u + gu);
                        }
                    }
                    Xold[q * BOX + pos] = val;
                }
            }
        }
        __syncthreads();

        // ---- 3. update all nodes
        for (int qd = threadIdx.x; qd < nquads; qd += blockDim.x) {
            const int vl = qd / quads_u, ql = qd - vl * quads_u;
            const int ul0 = ql * 4;
            const int gv = v0 + vl, gu0 = u0 + ul0;
            const int base = (vl + 1) * BOXU + ul0 + XPAD;
            const int nvalid = min(4, tu - ul0);
            // centres of this plane
            const float4 kp4 = *reinterpret_cast<const float4*>(Bc + base);
            const float4 sp4 = *reinterpret_cast<const float4*>(Bc + BOX + base);
            const float kp[4] = {kp4.x, kp4.y, kp4.z, kp4.w};
            const float sp[4] = {sp4.x, sp4.y, sp4.z, sp4.w};
            float a_p, a_0, a_up, a_dn;
            if (zmarch) { a_p = a_pl; a_0 = a_plprev; a_up = a_plprev; a_dn = a_plprev; }
            else {
                a_p = (gv <= kstar) ? 1.f : 0.f; a_0 = a_p;
                a_up = (gv - 1 <= kstar) ? 1.f : 0.f;     // upwind row for sv > 0
                a_dn = (gv + 1 <= kstar) ? 1.f : 0.f;     // upwind row for sv < 0
            }
            float xq[NSLOT][4];
            if (!dirichlet_plane) {
                float kf[3][6], sf[3][6];
#pragma unroll
                for (int r = 0; r < 3; ++r) {
                    const int rb = base + (r - 1) * BOXU;
                    const float4 kv = *reinterpret_cast<const float4*>(Bp + rb);
                    const float4 sv4 = *reinterpret_cast<const float4*>(Bp + BOX + rb);
                    kf[r][0] = Bp[rb - 1]; kf[r][1] = kv.x; kf[r][2] = kv.y; kf[r][3] = kv.z; kf[r][4] = kv.w; kf[r][5] = Bp[rb + 4];
                    sf[r][0] = Bp[BOX + rb - 1]; sf[r][1] = sv4.x; sf[r][2] = sv4.y; sf[r][3] = sv4.z; sf[r][4] = sv4.w; sf[r][5] = Bp[BOX + rb + 4];
                }
                if (J.ray[0].active) ray_quad_update<+1, +1>(kf, sf, kp, sp, Xold + 0 * BOX, base, BOXU, J.ray[0], a_p, a_0, a_up, xq[0]);
                if (J.ray[1].active) ray_quad_update<-1, +1>(kf, sf, kp, sp, Xold + 1 * BOX, base, BOXU, J.ray[1], a_p, a_0, a_up, xq[1]);
                if (J.ray[2].active) ray_quad_update<+1, -1>(kf, sf, kp, sp, Xold + 2 * BOX, base, BOXU, J.ray[2], a_p, a_0, a_dn, xq[2]);
                if (J.ray[3].active) ray_quad_update<-1, -1>(kf, sf, kp, sp, Xold + 3 * BOX, base, BOXU, J.ray[3], a_p, a_0, a_dn, xq[3]);
            }
            // Dirichlet nodes (not updated): I = S (upward, bottom) or I = 0 (downward, top)
            float qacc[4] = {0.f, 0.f, 0.f, 0.f};
            const bool edge_quad = (ul0 == 0) || (ul0 + 4 >= tu) || (vl == 0) || (vl == tv - 1);
#pragma unroll
            for (int q = 0; q < NSLOT; ++q) {
                const RayC& rc = J.ray[q];
                if (!rc.active) continue;
                const int su = (q & 1) ? -1 : 1, sv = (q & 2) ? -1 : 1;
                const bool dnode = zmarch ? dirichlet_plane : (gv == rc.dir_row);
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const float Stp = a_p * sp[j];
                    if (dnode) xq[q][j] = (rc.up ? sp[j] : 0.f) - Stp;
                    qacc[j] = fmaf(rc.wq, xq[q][j] - (sp[j] - Stp), qacc[j]);     // w_r (I - S)
                }
                // carried plane for the next step
                float* xn = Xnew + q * BOX + base;
                if (nvalid == 4) *reinterpret_cast<float4*>(xn) = make_float4(xq[q][0], xq[q][1], xq[q][2], xq[q][3]);
                else for (int j = 0; j < nvalid; ++j) xn[j] = xq[q][j];
                // publish edges / far faces
                if (edge_quad) {
                    const int ue = (su > 0) ? tu - 1 : 0, ve = (sv > 0) ? tv - 1 : 0;
                    const int gfu = (su > 0) ? n_u - 1 : 0, gfv = (sv > 0) ? n_v - 1 : 0;
                    for (int j = 0; j < nvalid; ++j) {
                        const int ul = ul0 + j, gu = gu0 + j;
                        if (ul == ue || vl == ve)
                            __stcg(J.Dg + ((size_t)(s & 1) * NSLOT + q) * plane_uv + (size_t)gv * n_u + gu, xq[q][j]);
                        if (gu == gfu)
                            __stcg(J.Gu + (((size_t)(pass & 1) * NSLOT + q) * n_m + m) * n_v + gv, xq[q][j]);
                        if (J.per_v && gv == gfv)
                            __stcg(J.Gv + (((size_t)(pass & 1) * NSLOT + q) * n_m + m) * n_u + gu, xq[q][j]);
                    }
                }
                // emergent intensity at the top node plane
                if (lastpass && rc.up && rc.itop >= 0 && Itop_b) {
                    const bool top = zmarch ? (m == n_m - 1) : (gv == J.nz - 1);
                    if (top) {
                        float* dst = Itop_b + (long long)rc.itop * J.it_sr + (zmarch ? (long long)gv : (long long)pl) * J.it_so;
                        for (int j = 0; j < nvalid; ++j) dst[(long long)(gu0 + j) * J.it_su] = xq[q][j] + a_p * sp[j];
                    }
                }
            }
            // fused J/Q reduction: Q += 4 pi kaprho_b sum_r w_r (I_r - S)
            if (lastpass) {
                float* qd_ = Qdst + (long long)pl * J.q_sm + (long long)gv * J.q_sv + gu0;
                for (int j = 0; j < nvalid; ++j) atomicAdd(qd_ + j, FOUR_PI * kp[j] * qacc[j]);
            }
        }
        __syncthreads();

        // ---- 4. publish progress, prefetch the plane after next
        if (threadIdx.x == 0) {
            __threadfence();
            st_release(my_progress, s + 1);
            if (s + 1 < nsteps) {
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                issue_load(s + 1);
            }
        }
    }
}

// =========================================================================== K_f
// Q[k][j][i] += QB[k][i][j]  (QB = heating of the x-march sweeps, stored y-fastest)
__global__ void __launch_bounds__(256) rts_finalize_kernel(float* Q, const float* QB, int nx, int ny, int nz)
{
    __shared__ float tile[32][33];
    const int tx = threadIdx.x, ty = threadIdx.y;
    const int i0 = blockIdx.x * 32, j0 = blockIdx.y * 32, k = blockIdx.z;
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        const int i = i0 + ty + 8 * r, j = j0 + tx;
        if (i < nx && j < ny) tile[ty + 8 * r][tx] = QB[((size_t)k * nx + i) * ny + j];
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        const int j = j0 + ty + 8 * r, i = i0 + tx;
        if (i < nx && j < ny) Q[((size_t)k * ny + j) * nx + i] += tile[tx][ty + 8 * r];
    }
}

}  // namespace rts
