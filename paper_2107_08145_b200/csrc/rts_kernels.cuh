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

constexpr int   NS = 2;             // rays per sweep job: su = +1 (slot 0) and su = -1 (slot 1)
constexpr int   XPAD = 4;           // ghost columns on each side of the unit-stride axis
constexpr int   NSTAGE = 3;         // depth of the coefficient-plane ring in shared memory
constexpr float LOG2E = 1.4426950408889634f;
constexpr float FOUR_PI = 12.566370614359172f;
constexpr float DTAU_SERIES = 0.05f; // below this the psi weights come from their series
constexpr double SIGMA_SB_D = 5.670374e-5;
constexpr double PI_D = 3.14159265358979323846;

struct alignas(16) RayC {
    float wx[4];      // bilinear weights of (u,v) (u-su,v) (u,v-sv) (u-su,v-sv); sum == 1 exactly
    float wk[4];      // 0.5*ds*wx  (opacity -> optical path)
    float kc;         // 0.5*ds
    float wq;         // quadrature weight
    int   active;
    int   up;         // mu_z > 0
    int   itop;       // index among the upward rays, or -1
    int   pad0, pad1, pad2;
};

// One sweep job: the rays that march along `march` in direction `dir` and whose transverse
// v-component has sign `sv` (at most one per u-sign), for one band.  Its tiles are full-width
// row bands [0,n_u) x [v0, v0+TV); tile t (in upwind-to-downwind order) depends only on tile
// t-1 of the same step range, so tiles form a one-way pipeline.
struct JobDesc {
    int march;        // 0: x, 1: y, 2: z  (axis the sweep marches along)
    int dir;          // +1 / -1 along the march axis
    int sv;           // +1 / -1 sign of the rays along v
    int band;
    int n_m, n_u, n_v;
    int TV, ntv;
    int per_v;        // v periodic (z-march: v = y) or bounded (x/y-march: v = z)
    int ticket_begin; // first ticket of this job; tile order = ticket order
    int npass;
    int nz;
    int q_in_B;       // heating goes to the y-fastest partial buffer (x-march)
    int pad0, pad1;
    RayC ray[NS];
    float* Hrow;      // [ntv][nsteps][NS][n_u4]  downwind edge row of every tile and step
    float* Gu;        // [ntv][2][n_m][NS][TV]    far-u column history (pass parity)
    int*   progress;  // [ntv] steps whose edge row is published
    const float* cbase; // coefficient array of this band: [2 fields][...] in layout A or B
    long long c_field, c_m, c_v;          // strides (floats) between fields, march planes, v rows
    long long c_off;                      // offset of (m = 0, v = 0, padded u = 0)
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
// TMA engine, non-tensor form: contiguous global -> shared copy completing on an mbarrier
__device__ __forceinline__ void bulk_load(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
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
// Persistent pipelined sweep.  CTAs take (job, tile) tasks from an in-order ticket counter.
// A task marches its row band plane by plane through all passes.  Per step:
//   - opacity / source rows of the plane are staged by the TMA engine (cp.async.bulk, 3-deep)
//   - the upwind ring row comes from the edge-row history of the upwind tile (same pass), or,
//     across the periodic seam in v, from the last tile's history one pass earlier; the ring
//     columns (periodic seam in u) from this tile's own far-column history of the previous
//     pass (Jacobi ghosts); pass 0 uses I = S
//   - every thread updates a 4 x 2 block of nodes for both rays from registers + shared memory
//   - the downwind edge row is appended to this tile's history and the step counter released
// Dependencies point one way (tile t needs tile t-1), so exchange latency only skews the
// pipeline; it never bounds the step rate.
// Carried quantity: X = I - a*S with a = 1 at levels k <= kstar (optically thick part, where
// J - S would cancel) and a = 0 above (thin part, where I << S would cancel).

// closed-form attenuation factors: em1 = 1 - e^-dt, wl = (1 - e^-dt)/dt
__device__ __forceinline__ void att_closed(float dt, float& em1, float& wl) {
    const float E = ex2_approx(-dt * LOG2E);
    em1 = 1.0f - E;
    wl = em1 * rcp_approx(dt);
}
// series below DTAU_SERIES: psi_p, psi_u directly (no cancellation), wl = 1 - psi_p, em1 = dt*wl
__device__ __forceinline__ void att_series(float dt, float& em1, float& wl, float& pu, float& pp) {
    pp = dt * (0.5f - dt * (1.0f / 6.0f - dt * (1.0f / 24.0f - dt * (1.0f / 120.0f))));
    pu = dt * (0.5f - dt * (1.0f / 3.0f - dt * (1.0f / 8.0f - dt * (1.0f / 30.0f))));
    wl = 1.0f - pp;
    em1 = dt * wl;
}

// One node row (4 consecutive nodes) of one ray with u-sign SU.
//   ko/so, ku/su_ : opacity / source of the previous plane on the node's own row and on its
//                   upwind row (6 values: columns ul0-1 .. ul0+4)
//   xo, xu        : carried quantity on the same two rows (6 values)
// REG 0: everything in the departure-carried part (a = 1); 1: all direct (a = 0); 2: mixed.
template <int SU, int REG>
__device__ __forceinline__ void ray_row_update(
    const float (&ko)[6], const float (&ku)[6], const float (&so)[6], const float (&su_)[6],
    const float (&xo)[6], const float (&xu)[6], const float (&kp)[4], const float (&sp)[4],
    const float4 wv, const float4 kv, const float kc,
    const float ap, const float a0, const float a1, const unsigned mask, float (&xp)[4])
{
    float Xu[4], dt[4];
    bool small = false;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const int c = j + 1, cs = j + 1 - SU;
        Xu[j] = wv.x * xo[c] + wv.y * xo[cs] + wv.z * xu[c] + wv.w * xu[cs];
        dt[j] = kc * kp[j] + kv.x * ko[c] + kv.y * ko[cs] + kv.z * ku[c] + kv.w * ku[cs];
        small |= dt[j] < DTAU_SERIES;
    }
    const bool any_small = __any_sync(mask, small);
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const int c = j + 1, cs = j + 1 - SU;
        float em1, wl, pu = 0.f, pp = 0.f;
        att_closed(dt[j], em1, wl);
        if (REG != 0) { pp = 1.0f - wl; pu = wl - 1.0f + em1; }
        if (any_small) {
            float e2, w2, pu2, pp2;
            att_series(dt[j], e2, w2, pu2, pp2);
            const bool sm = dt[j] < DTAU_SERIES;
            pp = sm ? pp2 : pp;
            pu = sm ? pu2 : pu;
            em1 = sm ? e2 : em1;
            wl = sm ? w2 : wl;
        }
        float v = fmaf(-Xu[j], em1, Xu[j]);
        if (REG == 0) {
            float dS = sp[j];
            dS = fmaf(-wv.x, so[c], dS); dS = fmaf(-wv.y, so[cs], dS);
            dS = fmaf(-wv.z, su_[c], dS); dS = fmaf(-wv.w, su_[cs], dS);
            v = fmaf(-dS, wl, v);
        } else if (REG == 1) {
            float Su = wv.x * so[c];
            Su = fmaf(wv.y, so[cs], Su); Su = fmaf(wv.z, su_[c], Su); Su = fmaf(wv.w, su_[cs], Su);
            v = fmaf(pu, Su, v);
            v = fmaf(pp, sp[j], v);
        } else {
            const float R0 = wv.x * so[c] + wv.y * so[cs];
            const float R1 = wv.z * su_[c] + wv.w * su_[cs];
            const float St = a0 * R0 + a1 * R1;
            const float Sh = (R0 + R1) - St;
            const float Stp = ap * sp[j];
            v = fmaf(-(Stp - St), wl, v);
            v = fmaf(pu, Sh, v);
            v = fmaf(pp, sp[j] - Stp, v);
        }
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

// 6 values of one box row around a quad: columns ul0-1 .. ul0+4.  The centre float4 comes from
// shared memory; the two side values come from the neighbouring lanes' float4 when those lanes
// hold the adjacent quads of the same row, else from shared memory.
__device__ __forceinline__ void load_row6(const float* __restrict__ row, bool left_lane_ok, bool right_lane_ok,
                                          float (&out)[6])
{
    const float4 v = *reinterpret_cast<const float4*>(row);
    float l = __shfl_up_sync(0xffffffffu, v.w, 1);
    float r = __shfl_down_sync(0xffffffffu, v.x, 1);
    if (!left_lane_ok) l = row[-1];
    if (!right_lane_ok) r = row[4];
    out[0] = l; out[1] = v.x; out[2] = v.y; out[3] = v.z; out[4] = v.w; out[5] = r;
}

template <int SV>
__device__ void run_task(const JobDesc& J, int t, unsigned char* smem_raw, uint64_t* mbar, int* s_flag,
                         float* __restrict__ Qa, float* __restrict__ Qb, float* __restrict__ Itop_all,
                         int* abortf)
{
    const int tid = threadIdx.x, nthr = blockDim.x, lane = tid & 31;
    const int n_u = J.n_u, n_v = J.n_v, n_m = J.n_m, TV = J.TV;
    const int n_u4 = (n_u + 3) & ~3;
    const int BOXU = n_u4 + 2 * XPAD, BOXV = TV + 2, BOX = BOXU * BOXV;
    const int b = (SV > 0) ? t : J.ntv - 1 - t;         // row-band index along v
    const int v0 = b * TV;
    const int tv = min(TV, n_v - v0);
    const bool zmarch = (J.march == 2);
    const int nsteps = n_m * J.npass;
    const int kstar = *J.kstar;
    float* const Qdst = J.q_in_B ? Qb : Qa;
    float* const Itop_b = Itop_all ? Itop_all + (long long)J.band * J.it_sb : nullptr;
    const RayC* const rays = J.ray;
    const bool has_up = (t > 0) || (J.per_v && J.ntv >= 1);     // an upwind tile (or the seam) exists
    const int t_up = (t > 0) ? t - 1 : J.ntv - 1;              // its tile index (seam: previous pass)
    const bool seam_up = (t == 0);

    // ---- shared memory: [NSTAGE][2][BOX] coefficient planes, [NS][BOX] carried quantity
    float* sm_f = reinterpret_cast<float*>(smem_raw);
    const int stage_floats = (2 * BOX + 31) & ~31;
    float* coef[NSTAGE];
#pragma unroll
    for (int i = 0; i < NSTAGE; ++i) coef[i] = sm_f + i * stage_floats;
    float* const X = sm_f + NSTAGE * stage_floats;
    // rows of the box that exist in memory (x/y-march: v = z is bounded; ghost rows stay zero)
    const int r_lo = (J.per_v || v0 > 0) ? 0 : 1;
    const int r_hi = (J.per_v || v0 + tv < n_v) ? tv + 1 : tv;  // inclusive box-row range [r_lo, r_hi]
    const uint32_t row_bytes = (uint32_t)(BOXU * sizeof(float));
    const uint32_t stage_bytes = 2u * (uint32_t)(r_hi - r_lo + 1) * row_bytes;

    for (int i = tid; i < NSTAGE * stage_floats + NS * BOX; i += nthr) sm_f[i] = 0.f;
    if (tid == 0) {
        for (int i = 0; i < NSTAGE; ++i) mbar_init(&mbar[i], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncthreads();

    auto issue_load = [&](int L) {           // L = load number; -1 is the plane "before" step 0
        const int m = (L < 0) ? n_m - 1 : (L % n_m);
        const int pl = (J.dir > 0) ? m : n_m - 1 - m;
        const int st = (L + NSTAGE) % NSTAGE;
        uint64_t* bar = &mbar[st];
        mbar_expect_tx(bar, stage_bytes);
        const float* src0 = J.cbase + J.c_off + (long long)pl * J.c_m;
        for (int f = 0; f < 2; ++f)
            for (int r = r_lo; r <= r_hi; ++r)
                bulk_load(coef[st] + f * BOX + r * BOXU, src0 + f * J.c_field + (long long)(v0 + r - 1) * J.c_v,
                          row_bytes, bar);
    };
    auto wait_load = [&](int L) {
        const int st = (L + NSTAGE) % NSTAGE;
        const uint32_t par = (uint32_t)(((L + 1) / NSTAGE) & 1);
        unsigned spins = 0;
        while (!mbar_try_wait(&mbar[st], par)) { if (spin_abort(abortf, spins)) break; }
    };
    if (tid == 0) {
        issue_load(-1);
        issue_load(0);
        if (nsteps > 1) issue_load(1);
    }

    // ---- this thread's blocks: 4 nodes x 2 rows; uniform trip count per warp
    const int quads_u = n_u4 >> 2;
    const int rpairs = (tv + 1) >> 1;
    const int nblk = quads_u * rpairs;
    const int nblk_pad = (nblk + 31) & ~31;

    int* const my_progress = J.progress + t;
    const int* const up_progress = J.progress + t_up;
    const size_t hrow_tile = (size_t)nsteps * NS * n_u4;
    float* const Hmine = J.Hrow + (size_t)t * hrow_tile;
    const float* const Hup = J.Hrow + (size_t)t_up * hrow_tile;
    float* const Gmine = J.Gu + (size_t)t * 2 * n_m * NS * TV;
    int known_up = 0;                                    // cached progress of the upwind tile

    const float4 w0 = *reinterpret_cast<const float4*>(rays[0].wx), k0 = *reinterpret_cast<const float4*>(rays[0].wk);
    const float4 w1 = *reinterpret_cast<const float4*>(rays[1].wx), k1 = *reinterpret_cast<const float4*>(rays[1].wk);
    const float kc0 = rays[0].kc, kc1 = rays[1].kc;
    const bool act0 = rays[0].active != 0, act1 = rays[1].active != 0;
    const int dir_row = (SV > 0) ? 0 : J.nz - 1;        // x/y-march: Dirichlet row of this job's rays
    const bool up_rays = zmarch ? (J.dir > 0) : (SV > 0);

    for (int s = 0; s < nsteps; ++s) {
        const int m = s % n_m;
        const int pass = s / n_m;
        const int pl = (J.dir > 0) ? m : n_m - 1 - m;
        const int plprev = pl - J.dir;
        const int mprev = (m == 0) ? n_m - 1 : m - 1;
        const float* const Bc = coef[s % NSTAGE];
        const float* const Bp = coef[(s + NSTAGE - 1) % NSTAGE];
        const float* const Sp_prev = Bp + BOX;
        const bool lastpass = (pass == J.npass - 1);
        const bool dirichlet_plane = zmarch && (m == 0);
        const float a_pl = (pl <= kstar) ? 1.f : 0.f;
        const float a_plprev = (plprev <= kstar) ? 1.f : 0.f;

        wait_load(s);
        if (s == 0) {
            wait_load(-1);
            if (!zmarch) {
                __syncthreads();
                // X^(0) = I^(0) - a S on the plane "before" step 0, ring included
                for (int idx = tid; idx < NS * BOX; idx += nthr) {
                    const int q = idx / BOX, pos = idx - q * BOX;
                    const int gv = v0 + pos / BOXU - 1;
                    const float Sv = Sp_prev[pos];
                    const float a = (gv <= kstar) ? 1.f : 0.f;
                    const float I0 = (gv == dir_row && !up_rays) ? 0.f : Sv;
                    X[idx] = I0 - a * Sv;
                }
            }
        } else if (!dirichlet_plane) {
            // ---- ring row from the upwind tile (or zero outside a bounded domain)
            const int need = seam_up ? s - n_m : s;     // steps the upwind tile must have published
            if (has_up && need > 0) {
                if (tid < 32 && known_up < need) {
                    unsigned spins = 0;
                    int v = 0;
                    while (true) {
                        if (lane == 0) v = ld_acquire(up_progress);
                        v = __shfl_sync(0xffffffffu, v, 0);
                        if (v >= need) break;
                        if (spin_abort(abortf, spins)) break;
                        __nanosleep(40);
                    }
                    if (lane == 0) *s_flag = v;
                }
                if (known_up < need) {
                    __syncthreads();
                    known_up = *s_flag;
                }
            }
            const int vr = (SV > 0) ? -1 : tv;          // ring row (local v) and its box row
            const int rowpos = (vr + 1) * BOXU + XPAD;
            const int gvr = v0 + vr;
            const bool row_outside = !J.per_v && (gvr < 0 || gvr >= n_v);
            const bool row_pass0 = seam_up && pass == 0;       // seam in v at pass 0: I^(0)
            const int hs = seam_up ? s - 1 - n_m : s - 1;      // step whose edge row we need
            for (int idx = tid; idx < NS * (n_u4 >> 2); idx += nthr) {
                const int q = idx / (n_u4 >> 2), c4 = idx - q * (n_u4 >> 2);
                float4 val = make_float4(0.f, 0.f, 0.f, 0.f);
                if (!row_outside) {
                    if (row_pass0) {
                        const float4 Sv = *reinterpret_cast<const float4*>(Sp_prev + rowpos + 4 * c4);
                        const float a = zmarch ? a_plprev : ((gvr <= kstar) ? 1.f : 0.f);
                        const bool dn = zmarch ? (mprev == 0) : false;
                        const float f = ((dn && !up_rays) ? 0.f : 1.f) - a;
                        val = make_float4(f * Sv.x, f * Sv.y, f * Sv.z, f * Sv.w);
                    } else {
                        val = __ldcg(reinterpret_cast<const float4*>(Hup + ((size_t)hs * NS + q) * n_u4) + c4);
                    }
                }
                float* dstp = X + q * BOX + rowpos + 4 * c4;
                if (4 * c4 + 4 <= n_u) *reinterpret_cast<float4*>(dstp) = val;
                else { const float vv[4] = {val.x, val.y, val.z, val.w}; for (int j = 0; j < n_u - 4 * c4; ++j) dstp[j] = vv[j]; }
            }
            // ---- ring columns (periodic seam in u): own far-column history of the previous pass,
            //      rows -1 .. tv (the ring-row corner belongs to the upwind tile's history)
            for (int idx = tid; idx < NS * (tv + 2); idx += nthr) {
                const int q = idx / (tv + 2), vl = idx - q * (tv + 2) - 1;
                const int su = q ? -1 : 1;
                const int ul = (su > 0) ? -1 : n_u;
                const int pos = (vl + 1) * BOXU + ul + XPAD;
                const int gv = v0 + vl;
                float val = 0.f;
                const bool outside = !J.per_v && (gv < 0 || gv >= n_v);
                if (!outside) {
                    if (pass == 0) {
                        const float Sv = Sp_prev[pos];
                        int gvw = gv; if (gvw < 0) gvw += n_v; else if (gvw >= n_v) gvw -= n_v;
                        const float a = zmarch ? a_plprev : ((gvw <= kstar) ? 1.f : 0.f);
                        const bool dn = zmarch ? (mprev == 0) : (gvw == dir_row);
                        val = ((dn && !up_rays) ? 0.f : Sv) - a * Sv;
                    } else {
                        const int pb = (pass - 1) & 1;
                        const int ufar = (su > 0) ? n_u - 1 : 0;
                        if (vl >= 0 && vl < tv) {
                            val = __ldcg(Gmine + (((size_t)pb * n_m + mprev) * NS + q) * TV + vl);
                        } else if (vl == vr && has_up) {
                            // corner (u and the row both upwind): far-u node of the upwind tile's edge
                            // row in pass p-1 -- step s-1 if the march plane itself wrapped (m == 0) or the
                            // row already is the v-seam (then the ring row is pass p-1 too), else s-1-n_m
                            const int hcs = seam_up ? s - 1 - n_m : (m == 0 ? s - 1 : s - 1 - n_m);
                            if (hcs >= 0) val = __ldcg(Hup + ((size_t)hcs * NS + q) * n_u4 + ufar);
                            else {
                                const float Sv = Sp_prev[pos];
                                int gvw = gv; if (gvw < 0) gvw += n_v; else if (gvw >= n_v) gvw -= n_v;
                                const float a = zmarch ? a_plprev : ((gvw <= kstar) ? 1.f : 0.f);
                                const bool dn = zmarch ? (mprev == 0) : (gvw == dir_row);
                                val = ((dn && !up_rays) ? 0.f : Sv) - a * Sv;
                            }
                        }
                    }
                }
                X[q * BOX + pos] = val;
            }
        }
        __syncthreads();

        // ---- update: every thread a 4 x 2 block, both rays; results stay in registers
        float xn[2][NS][4];     // [row of the pair][ray][node]
        int blk_base = 0, blk_vl = 0, blk_ul0 = 0;
        bool blk_valid = false;
        // (one block per thread per iteration; results of the LAST iteration are written after the
        //  barrier, earlier iterations are written straight away into a spare buffer -- not needed:
        //  the planner sizes tiles so that nblk <= blockDim.x)
        {
            const int e = tid;
            blk_valid = e < nblk;
            const int ec = blk_valid ? e : nblk - 1;
            const int rp = ec / quads_u, ql = ec - rp * quads_u;
            const int vl = rp * 2;
            blk_vl = vl; blk_ul0 = ql * 4;
            const int base = (vl + 1) * BOXU + ql * 4 + XPAD;   // box index of (row vl, node ul0)
            blk_base = base;
            const unsigned mask = 0xffffffffu;
            const bool l_ok = (lane > 0) && (ql > 0) && ((e - 1) / quads_u == rp) && (e < nblk);
            const bool r_ok = (lane < 31) && (ql < quads_u - 1) && (e + 1 < nblk);
            // rows of the previous plane: A = upwind row of the first node row, B, C
            //   SV > 0: node rows (vl, vl+1): A = vl-1, B = vl, C = vl+1 ; row 0 uses (B own, A upwind), row 1 uses (C own, B upwind)
            //   SV < 0: A = vl, B = vl+1, C = vl+2 ; row 0 uses (A own, B upwind), row 1 uses (B own, C upwind)
            const int rA = base + ((SV > 0) ? -BOXU : 0);
            const int rC = (SV > 0) ? rA + 2 * BOXU : min(rA + 2 * BOXU, (BOXV - 1) * BOXU + ql * 4 + XPAD);
            float kA[6], kB[6], kC[6], sA[6], sB[6], sC[6];
            if (!dirichlet_plane) {
                load_row6(Bp + rA, l_ok, r_ok, kA);
                load_row6(Bp + rA + BOXU, l_ok, r_ok, kB);
                load_row6(Bp + rC, l_ok, r_ok, kC);
                load_row6(Bp + BOX + rA, l_ok, r_ok, sA);
                load_row6(Bp + BOX + rA + BOXU, l_ok, r_ok, sB);
                load_row6(Bp + BOX + rC, l_ok, r_ok, sC);
            }
            const float4 kp0v = *reinterpret_cast<const float4*>(Bc + base);
            const float4 kp1v = *reinterpret_cast<const float4*>(Bc + base + BOXU);
            const float4 sp0v = *reinterpret_cast<const float4*>(Bc + BOX + base);
            const float4 sp1v = *reinterpret_cast<const float4*>(Bc + BOX + base + BOXU);
            const float kp[2][4] = {{kp0v.x, kp0v.y, kp0v.z, kp0v.w}, {kp1v.x, kp1v.y, kp1v.z, kp1v.w}};
            const float sp[2][4] = {{sp0v.x, sp0v.y, sp0v.z, sp0v.w}, {sp1v.x, sp1v.y, sp1v.z, sp1v.w}};
            // regime masks per node row
            float a_p[2], a_0[2], a_1[2];
#pragma unroll
            for (int r = 0; r < 2; ++r) {
                if (zmarch) { a_p[r] = a_pl; a_0[r] = a_plprev; a_1[r] = a_plprev; }
                else {
                    const int gv = v0 + vl + r;
                    a_p[r] = (gv <= kstar) ? 1.f : 0.f; a_0[r] = a_p[r];
                    a_1[r] = (gv - SV <= kstar) ? 1.f : 0.f;
                }
            }
            if (!dirichlet_plane) {
                const float asum = a_p[0] + a_0[0] + a_1[0] + a_p[1] + a_0[1] + a_1[1];
                const int reg = (asum == 6.f) ? 0 : (asum == 0.f) ? 1 : 2;
                const bool all0 = __all_sync(mask, reg == 0);
                const bool all1 = __all_sync(mask, reg == 1);
#pragma unroll
                for (int q = 0; q < NS; ++q) {
                    if (!(q ? act1 : act0)) continue;
                    const float* Xq = X + q * BOX;
                    float xA[6], xB[6], xC[6];
                    load_row6(Xq + rA, l_ok, r_ok, xA);
                    load_row6(Xq + rA + BOXU, l_ok, r_ok, xB);
                    load_row6(Xq + rC, l_ok, r_ok, xC);
                    const float4 wv = q ? w1 : w0, kv = q ? k1 : k0;
                    const float kc = q ? kc1 : kc0;
                    // row 0: own/upwind = (B, A) for SV > 0, (A, B) for SV < 0;  row 1: (C, B) / (B, C)
#define RTS_ROW(REG, R, KO, KU, SO, SU_, XO, XU)                                                        \
    if (q == 0) ray_row_update<+1, REG>(KO, KU, SO, SU_, XO, XU, kp[R], sp[R], wv, kv, kc, a_p[R], a_0[R], a_1[R], mask, xn[R][0]); \
    else        ray_row_update<-1, REG>(KO, KU, SO, SU_, XO, XU, kp[R], sp[R], wv, kv, kc, a_p[R], a_0[R], a_1[R], mask, xn[R][1]);
#define RTS_BLOCK(REG)                                                                                   \
    if (SV > 0) { RTS_ROW(REG, 0, kB, kA, sB, sA, xB, xA) RTS_ROW(REG, 1, kC, kB, sC, sB, xC, xB) }     \
    else        { RTS_ROW(REG, 0, kA, kB, sA, sB, xA, xB) RTS_ROW(REG, 1, kB, kC, sB, sC, xB, xC) }
                    if (all0) { RTS_BLOCK(0) } else if (all1) { RTS_BLOCK(1) } else { RTS_BLOCK(2) }
#undef RTS_BLOCK
#undef RTS_ROW
                }
            }
            // Dirichlet nodes (not updated): I = S (upward, bottom) or I = 0 (downward, top)
#pragma unroll
            for (int r = 0; r < 2; ++r) {
                const int gv = v0 + vl + r;
                const bool dn = dirichlet_plane || (!zmarch && gv == dir_row);
                if (dn) {
#pragma unroll
                    for (int q = 0; q < NS; ++q)
#pragma unroll
                        for (int j = 0; j < 4; ++j) xn[r][q][j] = (up_rays ? sp[r][j] : 0.f) - a_p[r] * sp[r][j];
                }
            }
            // heating and emergent intensity (last pass)
            if (lastpass && blk_valid) {
#pragma unroll
                for (int r = 0; r < 2; ++r) {
                    if (vl + r >= tv) continue;
                    const int gv = v0 + vl + r;
                    const int nvalid = min(4, n_u - blk_ul0);
                    float qa[4] = {0.f, 0.f, 0.f, 0.f};
                    const float shs = 1.0f - a_p[r];
#pragma unroll
                    for (int q = 0; q < NS; ++q) {
                        if (!(q ? act1 : act0)) continue;
                        const float wq = rays[q].wq;
#pragma unroll
                        for (int j = 0; j < 4; ++j) qa[j] = fmaf(wq, xn[r][q][j] - shs * sp[r][j], qa[j]);   // w_r (I - S)
                        if (up_rays && Itop_b && rays[q].itop >= 0) {
                            const bool top = zmarch ? (m == n_m - 1) : (gv == J.nz - 1);
                            if (top) {
                                float* dst = Itop_b + (long long)rays[q].itop * J.it_sr + (zmarch ? (long long)gv : (long long)pl) * J.it_so;
                                for (int j = 0; j < nvalid; ++j) dst[(long long)(blk_ul0 + j) * J.it_su] = xn[r][q][j] + a_p[r] * sp[r][j];
                            }
                        }
                    }
                    float* qd_ = Qdst + (long long)pl * J.q_sm + (long long)gv * J.q_sv + blk_ul0;
                    for (int j = 0; j < nvalid; ++j) atomicAdd(qd_ + j, FOUR_PI * kp[r][j] * qa[j]);
                }
            }
        }
        __syncthreads();

        // ---- write the carried plane, append the downwind edge row / far columns to the histories
        if (blk_valid) {
            const int ve = (SV > 0) ? tv - 1 : 0;          // downwind edge row (local)
#pragma unroll
            for (int r = 0; r < 2; ++r) {
                const int vl = blk_vl + r;
                if (vl >= tv) continue;
#pragma unroll
                for (int q = 0; q < NS; ++q) {
                    if (!(q ? act1 : act0)) continue;
                    const float4 v4 = make_float4(xn[r][q][0], xn[r][q][1], xn[r][q][2], xn[r][q][3]);
                    float* xw = X + q * BOX + blk_base + r * BOXU;
                    if (blk_ul0 + 4 <= n_u) *reinterpret_cast<float4*>(xw) = v4;
                    else for (int j = 0; j < n_u - blk_ul0; ++j) xw[j] = xn[r][q][j];
                    if (vl == ve)
                        __stcg(reinterpret_cast<float4*>(Hmine + ((size_t)s * NS + q) * n_u4) + (blk_ul0 >> 2), v4);
                    const int ufar = q ? 0 : n_u - 1;
                    if (ufar >= blk_ul0 && ufar < blk_ul0 + 4)
                        __stcg(Gmine + (((size_t)(pass & 1) * n_m + m) * NS + q) * TV + vl, xn[r][q][ufar - blk_ul0]);
                }
            }
        }
        __syncthreads();
        if (tid == 0) {
            __threadfence();
            st_release(my_progress, s + 1);
            if (s + 2 < nsteps) {
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                issue_load(s + 2);
            }
        }
        if ((s & 63) == 63) {       // uniform watchdog check
            if (tid == 0) s_flag[1] = *reinterpret_cast<const volatile int*>(abortf);
            __syncthreads();
            if (s_flag[1] != 0) break;
        }
    }
    __syncthreads();
    if (tid == 0)
        for (int i = 0; i < NSTAGE; ++i)
            asm volatile("mbarrier.inval.shared::cta.b64 [%0];" ::"r"(smem_u32(&mbar[i])) : "memory");
}

__global__ void __launch_bounds__(256, 2)
rts_sweep_kernel(const JobDesc* __restrict__ jobs, int njobs, int total_tickets, int* ticket_counter,
                 float* __restrict__ Qa, float* __restrict__ Qb, float* __restrict__ Itop_all, int* abortf)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ JobDesc J;
    __shared__ __align__(8) uint64_t mbar[NSTAGE];
    __shared__ int s_ticket;
    __shared__ int s_flag[2];
    while (true) {
        __syncthreads();
        if (threadIdx.x == 0) s_ticket = atomicAdd(ticket_counter, 1);
        __syncthreads();
        const int ticket = s_ticket;
        if (ticket >= total_tickets) break;
        int jid = 0;
        for (int q = 1; q < njobs; ++q)
            if (ticket >= jobs[q].ticket_begin) jid = q;
        {
            const int* src = reinterpret_cast<const int*>(jobs + jid);
            int* dst = reinterpret_cast<int*>(&J);
            for (int w = threadIdx.x; w < (int)(sizeof(JobDesc) / sizeof(int)); w += blockDim.x) dst[w] = src[w];
        }
        __syncthreads();
        const int t = ticket - J.ticket_begin;
        if (J.sv > 0) run_task<+1>(J, t, smem_raw, mbar, s_flag, Qa, Qb, Itop_all, abortf);
        else          run_task<-1>(J, t, smem_raw, mbar, s_flag, Qa, Qb, Itop_all, abortf);
        if (*reinterpret_cast<const volatile int*>(abortf) != 0) break;
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
