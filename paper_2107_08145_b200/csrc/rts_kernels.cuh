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
constexpr int   NSTAGE = 4;         // depth of the coefficient-plane ring in shared memory
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
// potentially blocking test: the warp is suspended by the hardware for up to ~`hint_ns`
// (no issue slots are burnt while the SM's other CTA computes)
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity, uint32_t hint_ns = 4000u) {
    uint32_t ok;
    asm volatile("{\n\t.reg .pred p;\n\t"
                 "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\t"
                 "selp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity), "r"(hint_ns) : "memory");
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
// "precision").  Writes kaprho_b, S_b in one layout per march axis, each with the rows of a
// sweep tile contiguous in memory (so that a tile's plane is one bulk copy per field):
//   layout Z  [b][f][nz][ny+2][PX]   x fastest (offset XPAD), rows y (offset 1, periodic ghost rows)
//   layout Y  [b][f][ny][nz+2][PX]   x fastest (offset XPAD), rows z (offset 1, zero pad rows)
//   layout X  [b][f][nx][nz+2][PY]   y fastest (offset XPAD), rows z (offset 1, zero pad rows)
// with periodic ghost columns along the fastest axis, and per-block partial sums of kaprho for K_k.
struct CoefParams {
    int nx, ny, nz, nb, nT, nP;
    double logT_min, inv_dT, logP_min, inv_dP;   // inv_d = (n-1)/(max-min)
    const float* logkappa;   // device [nb][nT][nP]
    const float* bandfrac;   // device [nb][nT]
    const float *rho, *T, *P;
    float* coefZ; float* coefY; float* coefX;
    int PX, PY;
    long long strideZ_f, strideY_f, strideX_f;   // field strides
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
    // periodic images of column i along x (layouts Z, Y)
    const int icols[3] = {i + XPAD, (i < XPAD) ? i + p.nx + XPAD : -1, (i >= p.nx - XPAD) ? i - p.nx + XPAD : -1};
    const bool zlo = (k == 0), zhi = (k == p.nz - 1);

    for (int b = 0; b < p.nb; ++b) {
        const float* L = p.logkappa + (size_t)b * p.nT * p.nP;
        const float* F = p.bandfrac + (size_t)b * p.nT;
        float* Z0 = p.coefZ + (size_t)(2 * b) * p.strideZ_f;  float* Z1 = Z0 + p.strideZ_f;
        float* Y0 = p.coefY + (size_t)(2 * b) * p.strideY_f;  float* Y1 = Y0 + p.strideY_f;
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
                const int jrows[3] = {j + 1, (j == 0) ? p.ny + 1 : -1, (j == p.ny - 1) ? 0 : -1};
#pragma unroll
                for (int c2 = 0; c2 < 3; ++c2) {
                    if (icols[c2] < 0) continue;
                    // layout Z: periodic ghost rows in y
#pragma unroll
                    for (int a2 = 0; a2 < 3; ++a2) {
                        if (jrows[a2] < 0) continue;
                        const size_t o = ((size_t)k * (p.ny + 2) + jrows[a2]) * p.PX + icols[c2];
                        Z0[o] = kr; Z1[o] = sr;
                    }
                    // layout Y: rows z, zero pad rows below / above the box
                    const size_t oy = ((size_t)j * (p.nz + 2) + (k + 1)) * p.PX + icols[c2];
                    Y0[oy] = kr; Y1[oy] = sr;
                    if (zlo) { Y0[oy - p.PX] = 0.f; Y1[oy - p.PX] = 0.f; }
                    if (zhi) { Y0[oy + p.PX] = 0.f; Y1[oy + p.PX] = 0.f; }
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
        // layout X: transposed write, coalesced along y
        float* X0 = p.coefX + (size_t)(2 * b) * p.strideX_f;  float* X1 = X0 + p.strideX_f;
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const int ii = i0 + ty + 8 * r, jj = j0 + tx;
            if (ii < p.nx && jj < p.ny) {
                const float kr = tile[0][tx][ty + 8 * r], sr = tile[1][tx][ty + 8 * r];
                const size_t rowoff = ((size_t)ii * (p.nz + 2) + (k + 1)) * p.PY;
                const int jc[3] = {jj + XPAD, (jj < XPAD) ? jj + p.ny + XPAD : -1, (jj >= p.ny - XPAD) ? jj - p.ny + XPAD : -1};
#pragma unroll
                for (int c2 = 0; c2 < 3; ++c2) {
                    if (jc[c2] < 0) continue;
                    X0[rowoff + jc[c2]] = kr; X1[rowoff + jc[c2]] = sr;
                    if (zlo) { X0[rowoff - p.PY + jc[c2]] = 0.f; X1[rowoff - p.PY + jc[c2]] = 0.f; }
                    if (zhi) { X0[rowoff + p.PY + jc[c2]] = 0.f; X1[rowoff + p.PY + jc[c2]] = 0.f; }
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

// One node row (4 consecutive nodes) of one ray with u-sign SU, in two phases so that the
// opacity rows are dead before the source / carried rows are loaded (register pressure).
//   ko/ku : opacity of the previous plane on the node's own row / upwind row (columns ul0-1..ul0+4)
template <int SU>
__device__ __forceinline__ void ray_row_dtau(const float (&ko)[6], const float (&ku)[6], const float (&kp)[4],
                                             const float4 kv, const float kc, float (&dt)[4])
{
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const int c = j + 1, cs = j + 1 - SU;
        dt[j] = kc * kp[j] + kv.x * ko[c] + kv.y * ko[cs] + kv.z * ku[c] + kv.w * ku[cs];
    }
}
//   so/su_ : source function on the same two rows; xo/xu: carried quantity
// REG 0: everything in the departure-carried part (a = 1); 1: all direct (a = 0); 2: mixed.
template <int SU, int REG>
__device__ __forceinline__ void ray_row_update(
    const float (&dt)[4], const float (&so)[6], const float (&su_)[6],
    const float (&xo)[6], const float (&xu)[6], const float (&sp)[4],
    const float4 wv, const float ap, const float a0, const float a1, const bool any_small, float (&xp)[4])
{
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const int c = j + 1, cs = j + 1 - SU;
        const float Xu = wv.x * xo[c] + wv.y * xo[cs] + wv.z * xu[c] + wv.w * xu[cs];
        float em1, wl;
        att_closed(dt[j], em1, wl);
        float pp = 1.0f - wl;
        if (any_small) {
            float e2, w2, pu2, pp2;
            att_series(dt[j], e2, w2, pu2, pp2);
            const bool sm = dt[j] < DTAU_SERIES;
            pp = sm ? pp2 : pp;
            em1 = sm ? e2 : em1;
            wl = sm ? w2 : wl;
        }
        const float pu = em1 - pp;                 // psi_u = (1-E)/dt - E = (1 - E) - psi_p
        float v = fmaf(-Xu, em1, Xu);
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

// watchdog for every wait loop: gives up after ~2^20 unsuccessful probes (seconds) and raises
// the device-side abort flag so that all CTAs drain instead of hanging the GPU
__device__ __forceinline__ bool spin_abort(const int* abortf, unsigned& spins, int code = 1)
{
    if ((++spins & 255u) == 0u) {
        if (*reinterpret_cast<const volatile int*>(abortf) != 0) return true;
        if (spins > (1u << 20)) { atomicCAS(const_cast<int*>(abortf), 0, code); return true; }
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

__device__ __forceinline__ void named_bar_sync(int id, int n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }
__device__ __forceinline__ void named_bar_arrive(int id, int n) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(n) : "memory"); }

#ifdef RTS_TRACE
__device__ unsigned long long g_trace[16384];
__device__ __forceinline__ unsigned long long gtime() { unsigned long long t; asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t)); return t; }
#define TRACE(slot) do { if (trace_on && s >= 200 && s < 264) g_trace[((s - 200) * 16) + (slot)] = gtime(); } while (0)
#else
#define TRACE(slot) do { } while (0)
#endif
constexpr int MAXC = 8;      // ring-column values per lane of the communication warp (NS * (TV + 2) <= 32 * MAXC)

__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}

template <int SV>
__device__ void run_task(const JobDesc& J, int t, unsigned char* smem_raw, uint64_t* mbar, int* s_flag,
                         float* __restrict__ Qa, float* __restrict__ Qb, float* __restrict__ Itop_all,
                         int* abortf)
{
    const int tid = threadIdx.x, nthr = blockDim.x, lane = tid & 31, warp = tid >> 5;
    const int NCW = (nthr >> 5) - 1;                    // compute warps; the last warp communicates
    const int ncomp = NCW * 32;
    const bool is_comm = (warp == NCW);
    const int n_u = J.n_u, n_v = J.n_v, n_m = J.n_m, TV = J.TV;
    const int n_u4 = (n_u + 3) & ~3;
    const int nq4 = n_u4 >> 2;
    const int BOXU = n_u4 + 2 * XPAD, BOXV = TV + 2, BOX = BOXU * BOXV;
    const int b = (SV > 0) ? t : J.ntv - 1 - t;         // row-band index along v
    const int v0 = b * TV;
    const int tv = min(TV, n_v - v0);
    const bool zmarch = (J.march == 2);
    const int npass = J.npass;
    const int nsteps = n_m * npass;
    const int kstar = *J.kstar;
    float* const Qdst = J.q_in_B ? Qb : Qa;
    float* const Itop_b = Itop_all ? Itop_all + (long long)J.band * J.it_sb : nullptr;
    const RayC* const rays = J.ray;
    const bool has_up = (t > 0) || J.per_v;             // an upwind tile (or the periodic seam) exists
    const int t_up = (t > 0) ? t - 1 : J.ntv - 1;
    const bool seam_up = (t == 0);
    const int dir_row = (SV > 0) ? 0 : J.nz - 1;        // x/y-march: Dirichlet row of this job's rays
    const bool up_rays = zmarch ? (J.dir > 0) : (SV > 0);
    const int vr = (SV > 0) ? -1 : tv;                  // ring row (local v)
    const int ve = (SV > 0) ? tv - 1 : 0;               // downwind edge row (local v)
    const bool row_outside = !J.per_v && (v0 + vr < 0 || v0 + vr >= n_v);

    // ---- shared memory: [NSTAGE][2][BOX] coefficient planes, [NS][BOX] carried quantity,
    //      [2][NS][BOXU] ring row of the carried quantity (double buffered, filled by TMA)
    float* sm_f = reinterpret_cast<float*>(smem_raw);
    const int stage_floats = (2 * BOX + 31) & ~31;
    const int x_floats = (NS * BOX + 31) & ~31;
    float* const X = sm_f + NSTAGE * stage_floats;
    float* const Ring = X + x_floats;                   // [2][NS][BOXU]  ring row (double buffered)
    uint64_t* const ringbar = mbar + NSTAGE;
    // the tile's rows (ring rows included; pad / ghost rows exist in memory) are contiguous
    const uint32_t field_bytes = (uint32_t)((tv + 2) * BOXU * sizeof(float));
    const uint32_t stage_bytes = 2u * field_bytes;

    for (int i = tid; i < NSTAGE * stage_floats + x_floats + 2 * NS * BOXU; i += nthr) sm_f[i] = 0.f;
    if (tid == 0) {
        for (int i = 0; i < NSTAGE + 2; ++i) mbar_init(&mbar[i], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        s_flag[1] = 0;
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncthreads();

    const float* const csrc0 = J.cbase + J.c_off + (long long)(v0 - 1) * J.c_v;
    auto issue_load = [&](int pl, int st) {             // one lane: the tile's plane, one copy per field
        uint64_t* bar = &mbar[st];
        mbar_expect_tx(bar, stage_bytes);
        float* dst = sm_f + st * stage_floats;
        const float* src = csrc0 + (long long)pl * J.c_m;
        bulk_load(dst, src, field_bytes, bar);
        bulk_load(dst + BOX, src + J.c_field, field_bytes, bar);
    };
    auto plane_of = [&](int m) { return (J.dir > 0) ? m : n_m - 1 - m; };
    if (tid == nthr - 32) {
        issue_load(plane_of(n_m - 1), NSTAGE - 1);      // load -1: the plane "before" step 0
        issue_load(plane_of(0), 0);
        if (nsteps > 1) issue_load(plane_of(1 % n_m), 1);
    }

    int* const my_progress = J.progress + t;
    const int* const up_progress = J.progress + t_up;
    const size_t hrow_tile = (size_t)nsteps * NS * n_u4;
    float* const Hmine = J.Hrow + (size_t)t * hrow_tile;
    const float* const Hup = J.Hrow + (size_t)t_up * hrow_tile;
    float* const Gmine = J.Gu + (size_t)t * 2 * n_m * NS * TV;

    // ---- step-invariant geometry of this thread's 4 x 2 block (compute warps)
    const int quads_u = nq4;
    const int nblk = quads_u * ((tv + 1) >> 1);
    const bool blk_valid = (!is_comm) && (tid < nblk);
    const int ec = min(tid, nblk - 1);
    const int rp = ec / quads_u, ql = ec - rp * quads_u;
    const int vl = rp * 2, ul0 = ql * 4;
    const int base = (vl + 1) * BOXU + ul0 + XPAD;      // box index of (row vl, node ul0)
    const bool l_ok = blk_valid && (lane > 0) && (ql > 0);
    const bool r_ok = blk_valid && (lane < 31) && (ql < quads_u - 1) && (tid + 1 < nblk);
    const int rA = base + ((SV > 0) ? -BOXU : 0);
    const int rB = rA + BOXU;
    const int rC = (SV > 0) ? rA + 2 * BOXU : min(rA + 2 * BOXU, (BOXV - 1) * BOXU + ul0 + XPAD);
    // rows of the carried quantity that are the ring row live in the Ring buffer
    const int ring_box_row = vr + 1;
    const bool ringA = (rA / BOXU == ring_box_row), ringB = (rB / BOXU == ring_box_row), ringC = (rC / BOXU == ring_box_row);
    const int ring_col = ul0 + XPAD;
    const bool row1_ok = (vl + 1 < tv);
    const bool full_u = (ul0 + 4 <= n_u);
    const int nvalid = min(4, n_u - ul0);
    float a_pi[2] = {0.f, 0.f}, a_1i[2] = {0.f, 0.f};   // x/y-march: masks depend on the row only
    if (!zmarch) {
#pragma unroll
        for (int r = 0; r < 2; ++r) {
            a_pi[r] = (v0 + vl + r <= kstar) ? 1.f : 0.f;
            a_1i[r] = (v0 + vl + r - SV <= kstar) ? 1.f : 0.f;
        }
    }
    float* const qbase = Qdst + (long long)(v0 + vl) * J.q_sv + ul0;

    // ---- communication warp, lanes 0 / 1: the corner of the ring row for ray 0 (u = -1) / ray 1 (u = n_u)
    const int cq = lane & 1;
    const int c_ringpos = cq * BOXU + (cq ? n_u : -1) + XPAD;           // position inside one Ring buffer
    const int c_hidx = cq * n_u4 + (cq ? 0 : n_u - 1);                   // far-u node in an edge-row record
    int c_gvw = v0 + vr; if (c_gvw < 0) c_gvw += n_v; else if (c_gvw >= n_v) c_gvw -= n_v;
    // ---- compute threads holding a far-u node store its periodic image (ring column) for the next
    //      step: the thread with u = n_u-1 writes ray 0's column u = -1, the thread with u = 0 writes
    //      ray 1's column u = n_u
    const bool seam_l = blk_valid && (ql == 0);
    const bool seam_r = blk_valid && (ul0 <= n_u - 1) && (n_u - 1 < ul0 + 4);
    const int colpos_l = (vl + 1) * BOXU + XPAD - 1;                      // box index of (row vl, u = -1)
    const int colpos_r = BOX + (vl + 1) * BOXU + n_u + XPAD;              // ray 1 array, (row vl, u = n_u)

    // ---- step 0 start-up (all threads): coefficient planes -1 and 0, X^(0)
    {
        unsigned spins = 0;
        while (!mbar_try_wait(&mbar[0], 0u)) { if (spin_abort(abortf, spins, 4)) break; }
        spins = 0;
        while (!mbar_try_wait(&mbar[NSTAGE - 1], 0u)) { if (spin_abort(abortf, spins, 5)) break; }
    }
    if (!zmarch) {
        // X^(0) = I^(0) - a S on the plane "before" step 0; its ring row goes to Ring[0]
        const float* Sp_prev = sm_f + (NSTAGE - 1) * stage_floats + BOX;
        for (int row = warp; row < BOXV; row += (nthr >> 5)) {
            const int gv = v0 + row - 1;
            const float a = (gv <= kstar) ? 1.f : 0.f;
            const float f = ((gv == dir_row && !up_rays) ? 0.f : 1.f) - a;
            for (int c = lane; c < BOXU; c += 32) {
                const float v = f * Sp_prev[row * BOXU + c];
                X[row * BOXU + c] = v;
                X[BOX + row * BOXU + c] = v;
                if (row == ring_box_row) { Ring[c] = v; Ring[BOXU + c] = v; }
            }
        }
    }
    __syncthreads();

    int m = 0, pass = 0;
    int stc = 0, stp = NSTAGE - 1;                      // stages of this step's and the previous plane
    uint32_t par_c = 0;                                 // parity of this step's stage barrier
    uint32_t ring_par = 0;                              // bit b: parity of ringbar[b] for its next use
#ifdef RTS_TRACE
    const bool trace_on = (J.ticket_begin + t == RTS_TRACE) && (lane == 0) && (warp == 0 || is_comm);
#endif
    for (int s = 0; s < nsteps; ++s) {
        const int pl = plane_of(m);
        const float* const Bc = sm_f + stc * stage_floats;
        const float* const Bp = sm_f + stp * stage_floats;
        const bool lastpass = (pass == npass - 1);
        const bool dirichlet_plane = zmarch && (m == 0);
        const float a_pl = (pl <= kstar) ? 1.f : 0.f;
        const float a_plprev = (pl - J.dir <= kstar) ? 1.f : 0.f;
        const int m1 = (m + 1 == n_m) ? 0 : m + 1;
        const int pass1 = (m + 1 == n_m) ? pass + 1 : pass;
        const int stn = (stc + 1 == NSTAGE) ? 0 : stc + 1;
        const int rb = s & 1;                           // ring buffer of this step

        if (is_comm) {
            // ================= communication warp =================
            TRACE(8);
            named_bar_sync(0, nthr);                    // B1(s): X(s-1) is in place
            TRACE(9);
            if (s > 0 && lane == 0) {                   // publish step s-1 (its edge row was stored before B1)
                __threadfence();
                st_release(my_progress, s);
            }
            TRACE(10);
            if (lane == 0 && s + 2 < nsteps) {          // coefficient planes two steps ahead
                const int m2 = (m1 + 1 == n_m) ? 0 : m1 + 1;
                int st2 = stc + 2; if (st2 >= NSTAGE) st2 -= NSTAGE;
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                issue_load(plane_of(m2), st2);          // last read in step s-1
            }
            // ---- ring row (+ corners) of step s+1 into the other ring buffer
            if (s + 1 < nsteps) {
                const bool ring_used = !(zmarch && m1 == 0);          // a Dirichlet plane reads no ring
                const bool row_pass0 = seam_up && pass1 == 0;
                const bool row_up = ring_used && has_up && !row_outside && !row_pass0;   // comes from the upwind tile
                const bool row_tma = row_up && (n_u4 == n_u);                             // (TMA needs whole float4 rows)
                const int hs = seam_up ? s - n_m : s;   // upwind step whose edge row feeds step s+1
                uint64_t* rbar = &ringbar[rb ^ 1];
                float* rdst = Ring + (rb ^ 1) * NS * BOXU;
                const float* Sp1 = Bc + BOX;            // source function of the plane before step s+1
                if (row_up) {
                    const int need = hs + 1;
                    unsigned spins = 0;
                    int v = 0;
                    while (true) {
                        if (lane == 0) v = ld_acquire(up_progress);
                        v = __shfl_sync(0xffffffffu, v, 0);
                        if (v >= need) break;
                        if (spin_abort(abortf, spins, 3 | (s << 4))) { if (lane == 0) s_flag[1] = 1; break; }
                        __nanosleep(40);
                    }
                    TRACE(11);
                }
                // corners: the periodic image in u of the upwind tile's far node, one pass earlier
                if (ring_used && !row_outside && lane < NS) {
                    const int hcs = seam_up ? s - n_m : (m1 == 0 ? s : s - n_m);
                    float val;
                    if (pass1 > 0 && has_up && hcs >= 0) val = __ldcg(Hup + (size_t)hcs * NS * n_u4 + c_hidx);
                    else {
                        const float Sv = Sp1[ring_box_row * BOXU + (cq ? n_u : -1) + XPAD];
                        const float a = zmarch ? a_pl : ((c_gvw <= kstar) ? 1.f : 0.f);
                        const bool dn = zmarch ? (m == 0) : (c_gvw == dir_row);
                        val = ((dn && !up_rays) ? 0.f : Sv) - a * Sv;
                    }
                    rdst[c_ringpos] = val;
                }
                if (row_tma) {
                    __syncwarp();
                    if (lane == 0) {
                        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                        mbar_expect_tx(rbar, (uint32_t)(NS * n_u4 * sizeof(float)));
                        const float* src = Hup + (size_t)hs * NS * n_u4;
                        bulk_load(rdst + XPAD, src, (uint32_t)(n_u4 * sizeof(float)), rbar);
                        bulk_load(rdst + BOXU + XPAD, src + n_u4, (uint32_t)(n_u4 * sizeof(float)), rbar);
                    }
                } else {
                    if (row_up) {                       // ragged width: plain copy of the valid nodes
                        const float* src = Hup + (size_t)hs * NS * n_u4;
                        for (int c = lane; c < n_u; c += 32) {
                            rdst[XPAD + c] = __ldcg(src + c);
                            rdst[BOXU + XPAD + c] = __ldcg(src + n_u4 + c);
                        }
                    } else if (ring_used && row_pass0 && !row_outside) {
                        // seam in v at pass 0: I^(0) of the plane before step s+1 (= this step's plane)
                        const float a_r = zmarch ? a_pl : ((c_gvw <= kstar) ? 1.f : 0.f);
                        const float f0 = ((zmarch && m == 0 && !up_rays) ? 0.f : 1.f) - a_r;
                        for (int c = lane; c < n_u; c += 32) {
                            const float v = f0 * Sp1[ring_box_row * BOXU + XPAD + c];
                            rdst[XPAD + c] = v; rdst[BOXU + XPAD + c] = v;
                        }
                    }
                    __syncwarp();
                    if (lane == 0) mbar_arrive(rbar);
                }
            }
            TRACE(12);
            TRACE(14);
        } else {
            // ================= compute warps =================
            TRACE(0);
            {
                unsigned spins = 0;
                while (!mbar_try_wait(&mbar[stc], par_c)) { if (spin_abort(abortf, spins, 2 | (s << 4))) break; }
                if (s > 0) {
                    spins = 0;
                    while (!mbar_try_wait(&ringbar[rb], (ring_par >> rb) & 1u)) { if (spin_abort(abortf, spins, 6 | (s << 4))) break; }
                    ring_par ^= (1u << rb);
                }
            }
            TRACE(1);
            named_bar_sync(0, nthr);                    // B1(s)
            TRACE(2);
            // u-seam threads: periodic image (previous pass) of the far-u node of their two rows for
            // step s+1; fetched now, stored in the write phase
            float gcol[2] = {0.f, 0.f};
            const bool seam_thr = seam_l || seam_r;
            const int sq = seam_r ? 0 : 1;               // (a 1-quad-wide band has both; ray 1 handled below)
            if (seam_thr && pass1 > 0 && m1 != 0 && pass1 < npass) {
                const float* g = Gmine + ((size_t)((pass1 - 1) & 1) * n_m + m) * NS * TV + vl;
                gcol[0] = __ldcg(g + sq * TV);
                if (row1_ok) gcol[1] = __ldcg(g + sq * TV + 1);
            }
            float gcol2[2] = {0.f, 0.f};
            const bool both = seam_l && seam_r;
            if (both && pass1 > 0 && m1 != 0 && pass1 < npass) {
                const float* g = Gmine + ((size_t)((pass1 - 1) & 1) * n_m + m) * NS * TV + vl;
                gcol2[0] = __ldcg(g + TV);
                if (row1_ok) gcol2[1] = __ldcg(g + TV + 1);
            }
            float xn[2][NS][4];
            float a_p[2], a_1[2];
#pragma unroll
            for (int r = 0; r < 2; ++r) {
                a_p[r] = zmarch ? a_pl : a_pi[r];
                a_1[r] = zmarch ? a_plprev : a_1i[r];
            }
            const float4 sp0v = *reinterpret_cast<const float4*>(Bc + BOX + base);
            const float4 sp1v = *reinterpret_cast<const float4*>(Bc + BOX + base + BOXU);
            const float sp[2][4] = {{sp0v.x, sp0v.y, sp0v.z, sp0v.w}, {sp1v.x, sp1v.y, sp1v.z, sp1v.w}};
            if (!dirichlet_plane) {
                // ---- phase 1: optical path of every (row, ray, node)
                float dt[2][NS][4];
                {
                    const float4 kp0v = *reinterpret_cast<const float4*>(Bc + base);
                    const float4 kp1v = *reinterpret_cast<const float4*>(Bc + base + BOXU);
                    const float kp[2][4] = {{kp0v.x, kp0v.y, kp0v.z, kp0v.w}, {kp1v.x, kp1v.y, kp1v.z, kp1v.w}};
                    float kA[6], kB[6], kC[6];
                    load_row6(Bp + rA, l_ok, r_ok, kA);
                    load_row6(Bp + rB, l_ok, r_ok, kB);
                    load_row6(Bp + rC, l_ok, r_ok, kC);
                    const float4 kv0 = *reinterpret_cast<const float4*>(rays[0].wk);
                    const float4 kv1 = *reinterpret_cast<const float4*>(rays[1].wk);
                    const float kc0 = rays[0].kc, kc1 = rays[1].kc;
                    if (SV > 0) {
                        ray_row_dtau<+1>(kB, kA, kp[0], kv0, kc0, dt[0][0]); ray_row_dtau<-1>(kB, kA, kp[0], kv1, kc1, dt[0][1]);
                        ray_row_dtau<+1>(kC, kB, kp[1], kv0, kc0, dt[1][0]); ray_row_dtau<-1>(kC, kB, kp[1], kv1, kc1, dt[1][1]);
                    } else {
                        ray_row_dtau<+1>(kA, kB, kp[0], kv0, kc0, dt[0][0]); ray_row_dtau<-1>(kA, kB, kp[0], kv1, kc1, dt[0][1]);
                        ray_row_dtau<+1>(kB, kC, kp[1], kv0, kc0, dt[1][0]); ray_row_dtau<-1>(kB, kC, kp[1], kv1, kc1, dt[1][1]);
                    }
                }
                bool small = false;
#pragma unroll
                for (int r = 0; r < 2; ++r)
#pragma unroll
                    for (int q = 0; q < NS; ++q)
#pragma unroll
                        for (int j = 0; j < 4; ++j) small |= dt[r][q][j] < DTAU_SERIES;
                const unsigned mask = 0xffffffffu;
                const bool any_small = __any_sync(mask, small);
                // ---- phase 2: source function and carried quantity
                float sA[6], sB[6], sC[6];
                load_row6(Bp + BOX + rA, l_ok, r_ok, sA);
                load_row6(Bp + BOX + rB, l_ok, r_ok, sB);
                load_row6(Bp + BOX + rC, l_ok, r_ok, sC);
                const float a00 = zmarch ? a_plprev : a_p[0], a01 = zmarch ? a_plprev : a_p[1];
                const float asum = a_p[0] + a00 + a_1[0] + a_p[1] + a01 + a_1[1];
                const int reg = (asum == 6.f) ? 0 : (asum == 0.f) ? 1 : 2;
                const bool all0 = __all_sync(mask, reg == 0);
                const bool all1 = __all_sync(mask, reg == 1);
#pragma unroll
                for (int q = 0; q < NS; ++q) {
                    if (!rays[q].active) {
#pragma unroll
                        for (int j = 0; j < 4; ++j) { xn[0][q][j] = 0.f; xn[1][q][j] = 0.f; }
                        continue;
                    }
                    const float* Xq = X + q * BOX;
                    const float* Rq = Ring + (rb * NS + q) * BOXU + ring_col;
                    float xA[6], xB[6], xC[6];
                    load_row6(ringA ? Rq : Xq + rA, l_ok, r_ok, xA);
                    load_row6(ringB ? Rq : Xq + rB, l_ok, r_ok, xB);
                    load_row6(ringC ? Rq : Xq + rC, l_ok, r_ok, xC);
                    const float4 wv = *reinterpret_cast<const float4*>(rays[q].wx);
#define RTS_ROW(REG, R, SO, SU_, XO, XU, A0)                                                             \
    if (q == 0) ray_row_update<+1, REG>(dt[R][0], SO, SU_, XO, XU, sp[R], wv, a_p[R], A0, a_1[R], any_small, xn[R][0]); \
    else        ray_row_update<-1, REG>(dt[R][1], SO, SU_, XO, XU, sp[R], wv, a_p[R], A0, a_1[R], any_small, xn[R][1]);
#define RTS_BLOCK(REG)                                                                                   \
    if (SV > 0) { RTS_ROW(REG, 0, sB, sA, xB, xA, a00) RTS_ROW(REG, 1, sC, sB, xC, xB, a01) }           \
    else        { RTS_ROW(REG, 0, sA, sB, xA, xB, a00) RTS_ROW(REG, 1, sB, sC, xB, xC, a01) }
                    if (all0) { RTS_BLOCK(0) } else if (all1) { RTS_BLOCK(1) } else { RTS_BLOCK(2) }
#undef RTS_BLOCK
#undef RTS_ROW
                }
            }
            TRACE(3);
            // Dirichlet nodes (not updated): I = S (upward, bottom) or I = 0 (downward, top)
#pragma unroll
            for (int r = 0; r < 2; ++r) {
                const bool dn = dirichlet_plane || (!zmarch && (v0 + vl + r) == dir_row);
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
                    if (r == 1 && !row1_ok) continue;
                    const int gv = v0 + vl + r;
                    const float4 kpv = *reinterpret_cast<const float4*>(Bc + base + r * BOXU);
                    const float kpq[4] = {kpv.x, kpv.y, kpv.z, kpv.w};
                    float qa[4] = {0.f, 0.f, 0.f, 0.f};
                    const float shs = 1.0f - a_p[r];
#pragma unroll
                    for (int q = 0; q < NS; ++q) {
                        if (!rays[q].active) continue;
                        const float wq = rays[q].wq;
#pragma unroll
                        for (int j = 0; j < 4; ++j) qa[j] = fmaf(wq, xn[r][q][j] - shs * sp[r][j], qa[j]);   // w_r (I - S)
                        if (up_rays && Itop_b && rays[q].itop >= 0) {
                            const bool top = zmarch ? (m == n_m - 1) : (gv == J.nz - 1);
                            if (top) {
                                float* dst = Itop_b + (long long)rays[q].itop * J.it_sr + (zmarch ? (long long)gv : (long long)pl) * J.it_so;
                                _Pragma("unroll") for (int j = 0; j < 4; ++j) if (j < nvalid) dst[(long long)(ul0 + j) * J.it_su] = xn[r][q][j] + a_p[r] * sp[r][j];
                            }
                        }
                    }
                    float* qd_ = qbase + (long long)pl * J.q_sm + (long long)r * J.q_sv;
                    _Pragma("unroll") for (int j = 0; j < 4; ++j) if (j < nvalid) atomicAdd(qd_ + j, FOUR_PI * kpq[j] * qa[j]);
                }
            }
            TRACE(4);
            named_bar_sync(1, ncomp);                   // every compute warp is done reading X
            TRACE(5);
            // ---- carried plane, edge-row and far-column histories
            if (blk_valid) {
#pragma unroll
                for (int r = 0; r < 2; ++r) {
                    if (r == 1 && !row1_ok) continue;
#pragma unroll
                    for (int q = 0; q < NS; ++q) {
                        if (!rays[q].active) continue;
                        const float4 v4 = make_float4(xn[r][q][0], xn[r][q][1], xn[r][q][2], xn[r][q][3]);
                        float* xw = X + q * BOX + base + r * BOXU;
                        if (full_u) *reinterpret_cast<float4*>(xw) = v4;
                        else { _Pragma("unroll") for (int j = 0; j < 4; ++j) if (j < nvalid) xw[j] = xn[r][q][j]; }
                        if (vl + r == ve)
                            __stcg(reinterpret_cast<float4*>(Hmine + ((size_t)s * NS + q) * n_u4) + ql, v4);
                        // far-u node of this ray (u = n_u-1 for ray 0, u = 0 for ray 1), static indexing only
                        if (q ? seam_l : seam_r) {
                            const float vf = q ? xn[r][1][0]
                                               : (nvalid == 4 ? xn[r][0][3] : nvalid == 3 ? xn[r][0][2] : nvalid == 2 ? xn[r][0][1] : xn[r][0][0]);
                            __stcg(Gmine + (((size_t)(pass & 1) * n_m + m) * NS + q) * TV + vl + r, vf);
                        }
                    }
                }
                // ring columns for step s+1 (periodic image in u, previous pass)
                if (seam_thr && s + 1 < nsteps) {
#pragma unroll
                    for (int side = 0; side < 2; ++side) {
                        const bool mine = side ? seam_l : seam_r;
                        if (!mine) continue;
                        const int q = side;
#pragma unroll
                        for (int r = 0; r < 2; ++r) {
                            if (r == 1 && !row1_ok) continue;
                            float val;
                            if (pass1 == 0) {              // previous pass = I^(0) of this step's plane
                                const int gv = v0 + vl + r;
                                const float Sv = Bc[BOX + (side ? colpos_r - BOX : colpos_l) + r * BOXU];
                                const float a = zmarch ? a_pl : ((gv <= kstar) ? 1.f : 0.f);
                                const bool dn = zmarch ? (m == 0) : (gv == dir_row);
                                val = ((dn && !up_rays) ? 0.f : Sv) - a * Sv;
                            } else if (m1 == 0) {          // pass boundary: this step's own far-u value
                                val = q ? xn[r][1][0]
                                        : (nvalid == 4 ? xn[r][0][3] : nvalid == 3 ? xn[r][0][2] : nvalid == 2 ? xn[r][0][1] : xn[r][0][0]);
                            } else {
                                val = (both && side) ? gcol2[r] : gcol[r];
                            }
                            X[(side ? colpos_r : colpos_l) + r * BOXU] = val;
                        }
                    }
                }
            }
            TRACE(6);
        }
        // advance the rotating indices
        m = m1; pass = pass1;
        stp = stc; stc = stn;
        if (stc == NSTAGE - 1) par_c ^= 1u;             // stage NSTAGE-1 already served load -1
        if ((s & 63) == 63) {                           // uniform watchdog check
            __syncthreads();
            if (s_flag[1] != 0 || *reinterpret_cast<const volatile int*>(abortf) != 0) { s_flag[1] = 1; }
            __syncthreads();
            if (s_flag[1] != 0) break;
        }
    }
    __syncthreads();
    if (tid == 0) {
        __threadfence();
        st_release(my_progress, nsteps);                // the last step's edge row
        for (int i = 0; i < NSTAGE + 2; ++i)
            asm volatile("mbarrier.inval.shared::cta.b64 [%0];" ::"r"(smem_u32(&mbar[i])) : "memory");
    }
}

__global__ void __launch_bounds__(256, 2)
rts_sweep_kernel(const JobDesc* __restrict__ jobs, int njobs, int total_tickets, int* ticket_counter,
                 float* __restrict__ Qa, float* __restrict__ Qb, float* __restrict__ Itop_all, int* abortf)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ JobDesc J;
    __shared__ __align__(8) uint64_t mbar[NSTAGE + 2];
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
