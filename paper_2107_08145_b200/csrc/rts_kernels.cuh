// rts_kernels.cuh -- device code of the RTS hot path (sm_100a), part 1: shared definitions,
// stage A and the small helper kernels.  The sweep kernel is in rts_sweep.cuh.
//
//   K_a  rts_coef_kernel    stage A  (paper's interpol())
//   K_k  rts_kstar_kernel   picks, per band pair, the height below which the sweep carries the
//                           departure I - S instead of I (precision device) and the
//                           optically thick levels the non-final passes may skip
//   K_b  rts_sweep_kernel   stages B-E (paper's integrate() + readbuf/writebuf/exchange with
//                           the box as its own neighbour + flux())
//   K_f  rts_finalize_kernel adds the x-march partial heating (stored y-fastest) into Q_rad
//   K_s  rts_cells_to_nodes_kernel / rts_nodes_to_cells_kernel   grid staggering
//
// Bands travel in PAIRS: every coefficient and every carried intensity is a float2 holding
// bands (2p, 2p+1) of one node, so that the whole update runs on packed fp32 pairs
// (fma.rn.f32x2: one issue slot for two bands).  An odd band count repeats the last band in
// the second half of the last pair; its results are never written.
//
// Shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <cuda.h>
#include <stdint.h>

namespace rts {

constexpr int   HALO = 4;           // ghost columns / rows around the periodic axes of the coefficient
                                    // layouts = halo allocation around a sweep tile
constexpr int   NSLOT = 4;          // rays per sweep unit: one per sign pair (su, sv)
constexpr int   NSTAGE_MAX = 3;     // deepest coefficient-plane ring in shared memory
constexpr int   KMAX = 4;           // most steps between two halo exchanges (<= HALO)
constexpr float LOG2E = 1.4426950408889634f;
constexpr float FOUR_PI = 12.566370614359172f;
constexpr float DTAU_SERIES = 0.05f; // below this the psi weights come from their series
constexpr double SIGMA_SB_D = 5.670374e-5;
constexpr double PI_D = 3.14159265358979323846;

// One ray of a sweep unit.  (u, v) are the transverse axes of the march; su, sv the signs of
// the ray along them.  Slot s of a unit holds a ray with su = (s & 1 ? -1 : +1),
// sv = (s & 2 ? -1 : +1).
struct alignas(16) RayC {
    float w[4];       // bilinear weights, sum == 1 exactly: (upwind v row, its u-side neighbour, the node's
                      // own v row, its u-side neighbour) of the previous plane
    float kc;         // 0.5*ds  (opacity sum -> optical path)
    float wq;         // quadrature weight
    int   active;
    int   up;         // mu_z > 0
    int   itop;       // index among the upward rays, or -1
    float mu[3];      // unit direction of photon travel (x, y, z): radiative flux
};

// One sweep unit: the (at most four) rays that march along `march` in direction `dir`, for one
// band pair.  The transverse plane is cut into ntu x ntv tiles of WU x WV nodes; one CTA owns one
// tile for the whole march (all planes, all passes).  Tiles exchange K-deep halos every K steps
// through Xex and meet at `barrier`; the periodic seams read the previous pass from Gu.
struct UnitDesc {
    int march;        // 0: x, 1: y, 2: z  (axis the sweep marches along)
    int dir;          // +1 / -1 along the march axis
    int pair;         // band pair: bands 2*pair, 2*pair + 1
    int per_v;        // v periodic (z-march: v = y) or bounded (x/y-march: v = z)
    int n_m, n_u, n_v, n_u2;               // n_u2 = n_u rounded up to even (row pitch of Xex / Gu, nodes)
    int WU, WV, ntu, ntv;
    int K, npass, ticket_begin, ntiles;
    int nz, q_in_B, qvec, nstage;          // qvec: heating rows are 16-byte aligned (vector reductions)
    int ng, gsu0, nband_ok, RC;            // ray groups (same su) of this unit: 2 (su = +1, -1) or 1 (su = gsu0);
    int xflag, pad0_;                      // 1: tagged exchange (every ray of the unit has its opposite ray in the unit)
                                           // nband_ok: bands of the pair that exist (1 or 2); RC: rows per strip
    RayC ray[NSLOT];
    float* Xex;       // [2][NSLOT][n_v][n_u2] x 16 bytes: carried planes at block ends (strips only), per node and
                      // band one 64-bit word (value, tag of the block that wrote it)
    float* Gu;        // float2 [2][n_m][NSLOT*n_v + NSLOT*n_u2]  per pass parity and plane: far-u column
                      //                                of every slot, then (per_v only) far-v row of every slot
    float* Qpart;     // [N] heating of this unit alone, in the unit's own layout (x- or y-fastest): every node is
                      // written exactly once per solve, the units are summed in a fixed order by rts_finalize_kernel
    float* Fpart;     // [3][N] radiative flux of this unit alone (same layout), or null
    int*   barrier;   // arrivals of this unit's tiles (monotonic)
    float* Lp;        // float2 [NSLOT][n_v][n_u2]: x/y-march, error-controlled mode: the last plane of the previous pass
    unsigned* errw;   // [NSLOT][4] error words of this unit (error-controlled mode), see TaskShared::errs
    const int* kstar; // device: switch height of this band pair
    const int* mthick;// device: thick level pairs from the bottom of this band pair (z-march plane skipping)
    long long q_sm, q_sv;                 // heating strides along (march, v); u stride 1
    long long it_su, it_so, it_sr, it_sb; // I_top strides along u, march-or-v axis, ray, band
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
// "precision").  Writes (kaprho, S) of every band pair as float2 per node in two layouts, both
// with HALO periodic images on each side of every periodic axis that a sweep tile can reach across:
//   layout A  [pair][f][nz][ny+2H][PX] float2   x fastest (offset H), rows y (offset H)   z- and y-march
//   layout B  [pair][f][nz][nx][PY]    float2   y fastest (offset H)                       x-march
// plus per-block partial sums / minima of kaprho per band for K_k.
struct CoefParams {
    int nx, ny, nz, nb, nT, nP;
    double logT_min, inv_dT, logP_min, inv_dP;   // inv_d = (n-1)/(max-min)
    const float* logkappa;   // device [nb][nT][nP]
    const float* bandfrac;   // device [nb][nT]
    const float *rho, *T, *P;
    float* coefA; float* coefB;
    int PX, PY, PYR;                             // padded row lengths / row count (nodes)
    long long strideA_n, strideB_n;              // field strides (nodes)
    double* ksum;            // [nb][nz][nblk] partial sums (nblk = gridDim.x*gridDim.y), or null
    float* kmin;             // [nb][nz][nblk] partial minima of kaprho (with ksum)
    float* plain_k; float* plain_s;              // optional [nb][N] outputs (rts_coefficients)
    int k0;                                      // first level of this launch (gridDim.z levels: rts_solve_host feeds slabs)
};

// 4 CTAs per SM (64 registers, ~200 bytes of spills into an L1 this kernel does not otherwise use): the kernel is bound by
// issue latency (table look-ups, fp64 log10 / exp10 chains), and 32 warps hide it better than 16: 1.42 -> 1.19 ms at 288^3 x 4
__global__ void __launch_bounds__(256, 4) rts_coef_kernel(const CoefParams p)
{
    __shared__ float2 tile[2][32][33];
    __shared__ double red[2][8];
    __shared__ float redm[2][8];
    const int tx = threadIdx.x, ty = threadIdx.y;
    const int i0 = blockIdx.x * 32, j0 = blockIdx.y * 32, k = p.k0 + blockIdx.z;
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
    const int cA0 = (i + HALO) % p.nx;            // first padded column of layout A congruent to i
    const int npair = (p.nb + 1) >> 1;

    for (int pr = 0; pr < npair; ++pr) {
        float2* A0 = reinterpret_cast<float2*>(p.coefA) + (size_t)(2 * pr) * p.strideA_n;
        float2* A1 = A0 + p.strideA_n;
        double part[2] = {0.0, 0.0};
        float pmin[2] = {3.0e38f, 3.0e38f};
        const int nbe = (2 * pr + 1 < p.nb) ? 2 : 1;
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            float kr[2] = {0.f, 0.f}, sr[2] = {0.f, 0.f};
            if (ok[r]) {
                const int a = it_[r], c = ip_[r];
                const double t = t_[r], u = u_[r];
                const int j = j0 + ty + 8 * r;
                for (int e = 0; e < nbe; ++e) {
                    const int b = 2 * pr + e;
                    const float* L = p.logkappa + (size_t)b * p.nT * p.nP;
                    const float* F = p.bandfrac + (size_t)b * p.nT;
                    const double l00 = (double)L[(size_t)a * p.nP + c], l10 = (double)L[(size_t)(a + 1) * p.nP + c];
                    const double l01 = (double)L[(size_t)a * p.nP + c + 1], l11 = (double)L[(size_t)(a + 1) * p.nP + c + 1];
                    const double lk = (1.0 - t) * (1.0 - u) * l00 + t * (1.0 - u) * l10 + (1.0 - t) * u * l01 + t * u * l11;
                    const double fb = (1.0 - t) * (double)F[a] + t * (double)F[a + 1];
                    const double kd = exp10(lk) * rho_[r];
                    kr[e] = (float)kd;
                    sr[e] = (float)(fb * planck[r]);
                    part[e] += kd;
                    pmin[e] = fminf(pmin[e], kr[e]);
                    if (p.plain_k) {
                        const long long n = ((long long)k * p.ny + j) * p.nx + i;
                        p.plain_k[(size_t)b * N + n] = kr[e];
                        p.plain_s[(size_t)b * N + n] = sr[e];
                    }
                }
                if (nbe == 1) { kr[1] = kr[0]; sr[1] = sr[0]; }     // odd band count: the last band twice
                // layout A: every periodic image of (i, j) inside the padded plane
                const float2 kv = make_float2(kr[0], kr[1]), sv = make_float2(sr[0], sr[1]);
                for (int row = (j + HALO) % p.ny; row < p.PYR; row += p.ny) {
                    const size_t ro = ((size_t)k * p.PYR + row) * p.PX;
                    for (int col = cA0; col < p.PX; col += p.nx) { A0[ro + col] = kv; A1[ro + col] = sv; }
                }
            }
            tile[0][ty + 8 * r][tx] = make_float2(kr[0], kr[1]);
            tile[1][ty + 8 * r][tx] = make_float2(sr[0], sr[1]);
        }
        // block sums / minima of kaprho per band (deterministic order)
        if (p.ksum) {
#pragma unroll
            for (int e = 0; e < 2; ++e) {
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) {
                    part[e] += __shfl_xor_sync(0xffffffffu, part[e], o);
                    pmin[e] = fminf(pmin[e], __shfl_xor_sync(0xffffffffu, pmin[e], o));
                }
                if (tx == 0) { red[e][ty] = part[e]; redm[e][ty] = pmin[e]; }
            }
        }
        __syncthreads();
        if (p.ksum && tx == 0 && ty < nbe) {
            double s = 0.0;
            float mn = 3.0e38f;
            for (int w = 0; w < 8; ++w) { s += red[ty][w]; mn = fminf(mn, redm[ty][w]); }
            const int nblk = gridDim.x * gridDim.y;
            const size_t o = ((size_t)(2 * pr + ty) * p.nz + k) * nblk + blockIdx.y * gridDim.x + blockIdx.x;
            p.ksum[o] = s;
            p.kmin[o] = mn;
        }
        // layout B: transposed write, coalesced along y
        float2* B0 = reinterpret_cast<float2*>(p.coefB) + (size_t)(2 * pr) * p.strideB_n;
        float2* B1 = B0 + p.strideB_n;
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const int ii = i0 + ty + 8 * r, jj = j0 + tx;
            if (ii < p.nx && jj < p.ny) {
                const float2 kv = tile[0][tx][ty + 8 * r], sv = tile[1][tx][ty + 8 * r];
                const size_t ro = ((size_t)k * p.nx + ii) * p.PY;
                for (int col = (jj + HALO) % p.ny; col < p.PY; col += p.ny) { B0[ro + col] = kv; B1[ro + col] = sv; }
            }
        }
        __syncthreads();
    }
}

// =========================================================================== K_k
// Per band: kstar_b = highest level k whose horizontally averaged optical depth from the top,
// tau(k) = sum_{k' >= k} <kaprho_b>(k') dz, is >= tau_switch (-1 if none).
// mthick_b[2] = number of consecutive level pairs (k-1, k), k = 1, 2, ..., from the bottom on which every
// optical path of a z-march ray exceeds DTAU_SKIP: kc * (min kaprho(k-1) + min kaprho(k)) > DTAU_SKIP bounds
// dtau = kc*(kaprho_p + sum_n w_n*kaprho_n) from below (kc = smallest half path of the z-march rays).
// mthick_b[0], [1] = number of consecutive levels from the bottom on which every optical path of an x- / y-march
// ray exceeds DTAU_SKIP (the stencil of such a node lies on its own level and the one below or above:
// 2*kc*min over the three levels bounds dtau).  There the approximate exp underflows to exactly 0 and the
// update does not depend on the carried intensity (rts_sweep.cuh).  One block per band pair; the pair takes the higher switch height and the
// smaller thick counts of its two bands (both bands ride in one float2).
constexpr float DTAU_SKIP = 88.5f;
struct KstarParams {
    const double* ksum; const float* kmin;
    int nb, nz, nblk;
    double inv_nxy, dz, tau_switch;
    double kc[3];            // per march axis (0: no such ray / shortcut off)
    int* kstar_pair;         // [npair]
    int* mthick_pair;        // [npair][3]
    int* mthick_band;        // [nb][3]    (reporting)
    double* lev;             // scratch [nb][2][nz]
};
__global__ void __launch_bounds__(1024) rts_kstar_kernel(const KstarParams p)
{
    __shared__ int sh_ks[2], sh_mt[2][3];
    const int pr = blockIdx.x;
    const int nz = p.nz, nblk = p.nblk;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
    const int nbe = (2 * pr + 1 < p.nb) ? 2 : 1;
    for (int e = 0; e < nbe; ++e) {
        const int b = 2 * pr + e;
        double* L = p.lev + (size_t)b * 2 * nz;
        double* M = L + nz;
        for (int k = warp; k < nz; k += nw) {             // level sums (fixed order) and level minima
            const double* q = p.ksum + ((size_t)b * nz + k) * nblk;
            const float* qm = p.kmin + ((size_t)b * nz + k) * nblk;
            double s = 0.0;
            float mn = 3.0e38f;
            for (int w = lane; w < nblk; w += 32) { s += q[w]; mn = fminf(mn, qm[w]); }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) { s += __shfl_xor_sync(0xffffffffu, s, o); mn = fminf(mn, __shfl_xor_sync(0xffffffffu, mn, o)); }
            if (lane == 0) { L[k] = s; M[k] = (double)mn; }
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            double tau = 0.0;
            int ks = -1;
            for (int k = nz - 1; k >= 0; --k) {
                tau += L[k] * p.inv_nxy * p.dz;
                if (tau >= p.tau_switch) { ks = k; break; }
            }
            sh_ks[e] = ks;
            for (int a = 0; a < 3; ++a) {
                int m = 0;
                if (p.kc[a] > 0.0) {
                    if (a == 2) {
                        for (int k = 1; k < nz; ++k) {
                            if (p.kc[a] * (M[k - 1] + M[k]) > (double)DTAU_SKIP) m = k; else break;
                        }
                    } else {
                        // x- / y-march: levels 0 .. m-1 are thick for upward and downward rays alike
                        for (int k = 0; k < nz; ++k) {
                            const double mn = fmin(M[k], fmin(M[max(k - 1, 0)], M[min(k + 1, nz - 1)]));
                            if (2.0 * p.kc[a] * mn > (double)DTAU_SKIP) m = k + 1; else break;
                        }
                    }
                }
                sh_mt[e][a] = m;
                p.mthick_band[b * 3 + a] = m;
            }
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        p.kstar_pair[pr] = (nbe == 2) ? max(sh_ks[0], sh_ks[1]) : sh_ks[0];
        for (int a = 0; a < 3; ++a)
            p.mthick_pair[pr * 3 + a] = (nbe == 2) ? min(sh_mt[0][a], sh_mt[1][a]) : sh_mt[0][a];
    }
}

// =========================================================================== K_f
// Q[k][j][i] = sum over the sweep units, in unit order, of the unit's partial heating (deterministic: no
// atomics anywhere on the heating path).  The partials of the x-march units are stored y-fastest
// ([nz][nx][ny]) and are transposed through shared memory.  nf fields per unit (1: Q; 4: Q, Fx, Fy, Fz):
// part[u] points at the unit's first field, the fields are N floats apart; out[f] may be null.
struct FinalizeParams {
    const float* const* part;   // device [nunits] partial buffers: the x-fastest ones first, then the y-fastest ones
    int nplain;                 // number of x-fastest buffers
    int nunits, nf;
    int nx, ny, nz;
    float* out[4];
};
__global__ void __launch_bounds__(256) rts_finalize_kernel(const FinalizeParams p)
{
    __shared__ float tile[32][33];
    const int tx = threadIdx.x, ty = threadIdx.y;
    const int i0 = blockIdx.x * 32, j0 = blockIdx.y * 32, k = blockIdx.z;
    const size_t N = (size_t)p.nx * p.ny * p.nz;
    const int ii = i0 + tx;
    for (int f = 0; f < p.nf; ++f) {
        if (!p.out[f]) continue;
        float acc[4] = {0.f, 0.f, 0.f, 0.f};
        // x-fastest partials, four buffers' loads in flight together (the sum stays in buffer order)
        int u = 0;
        for (; u + 4 <= p.nplain; u += 4) {
            float v[4][4];
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const float* src = p.part[u + q] + (size_t)f * N;
#pragma unroll
                for (int r = 0; r < 4; ++r) {
                    const int j = j0 + ty + 8 * r;
                    v[q][r] = (ii < p.nx && j < p.ny) ? __ldcs(src + ((size_t)k * p.ny + j) * p.nx + ii) : 0.f;
                }
            }
#pragma unroll
            for (int q = 0; q < 4; ++q)
#pragma unroll
                for (int r = 0; r < 4; ++r) acc[r] += v[q][r];
        }
        for (; u < p.nplain; ++u) {
            const float* src = p.part[u] + (size_t)f * N;
#pragma unroll
            for (int r = 0; r < 4; ++r) {
                const int j = j0 + ty + 8 * r;
                if (ii < p.nx && j < p.ny) acc[r] += __ldcs(src + ((size_t)k * p.ny + j) * p.nx + ii);
            }
        }
        // y-fastest partials (x-march units), transposed through shared memory; two buffers' loads in flight
        for (; u < p.nunits; u += 2) {
            const bool two = (u + 1 < p.nunits);
            const float* s0 = p.part[u] + (size_t)f * N;
            const float* s1 = two ? p.part[u + 1] + (size_t)f * N : s0;
            float a[4], b[4];
#pragma unroll
            for (int r = 0; r < 4; ++r) {
                const int i = i0 + ty + 8 * r, j = j0 + tx;
                const bool in = (i < p.nx && j < p.ny);
                const size_t o = ((size_t)k * p.nx + i) * p.ny + j;
                a[r] = in ? __ldcs(s0 + o) : 0.f;
                b[r] = (in && two) ? __ldcs(s1 + o) : 0.f;
            }
            __syncthreads();
#pragma unroll
            for (int r = 0; r < 4; ++r) tile[ty + 8 * r][tx] = a[r];
            __syncthreads();
#pragma unroll
            for (int r = 0; r < 4; ++r) acc[r] += tile[tx][ty + 8 * r];
            if (two) {
                __syncthreads();
#pragma unroll
                for (int r = 0; r < 4; ++r) tile[ty + 8 * r][tx] = b[r];
                __syncthreads();
#pragma unroll
                for (int r = 0; r < 4; ++r) acc[r] += tile[tx][ty + 8 * r];
            }
        }
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const int j = j0 + ty + 8 * r;
            if (ii < p.nx && j < p.ny) p.out[f][((size_t)k * p.ny + j) * p.nx + ii] = acc[r];
        }
    }
}

// =========================================================================== K_d (NEXT #2)
// Flux-divergence heating and its blend with the J - S form (paper's Flux; reading R21):
//   Qdiv = -(dFx/dx + dFy/dy + dFz/dz), central differences on the node grid, periodic in x and y, one-sided
//   on the bottom and top node planes;  Qblend = w Q_J + (1 - w) Qdiv with w(k) = exp(-taubar(k)/tau0),
//   taubar(k) = horizontally averaged optical depth of band 0 from the top down to level k (K_k's level sums).
// Any of Qdiv / Qblend may be null.
__global__ void __launch_bounds__(256) rts_fluxdiv_kernel(const float* __restrict__ F, const float* __restrict__ QJ,
                                                          float* __restrict__ Qdiv, float* __restrict__ Qblend,
                                                          const double* __restrict__ lev0, int nx, int ny, int nz,
                                                          float hx, float hy, float hz, double inv_nxy, double dz, double tau0)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y, k = blockIdx.z;
    if (i >= nx) return;
    const size_t N = (size_t)nx * ny * nz, row = ((size_t)k * ny + j) * nx;
    const int ip = (i + 1 == nx) ? 0 : i + 1, im = (i == 0) ? nx - 1 : i - 1;
    const int jp = (j + 1 == ny) ? 0 : j + 1, jm = (j == 0) ? ny - 1 : j - 1;
    const float dfx = (F[row + ip] - F[row + im]) * (0.5f / hx);
    const float dfy = (F[N + ((size_t)k * ny + jp) * nx + i] - F[N + ((size_t)k * ny + jm) * nx + i]) * (0.5f / hy);
    const int kp = min(k + 1, nz - 1), km = max(k - 1, 0);
    const float dfz = (F[2 * N + ((size_t)kp * ny + j) * nx + i] - F[2 * N + ((size_t)km * ny + j) * nx + i]) / (hz * (float)(kp - km));
    const float qd = -(dfx + dfy + dfz);
    if (Qdiv) Qdiv[row + i] = qd;
    if (Qblend) {
        double tau = 0.0;
        for (int kk = nz - 1; kk >= k; --kk) tau += lev0[kk] * inv_nxy * dz;
        const float w = (float)exp(-tau / tau0);
        Qblend[row + i] = w * QJ[row + i] + (1.f - w) * qd;
    }
}

// =========================================================================== K_s (NEXT #1)
// Grid staggering (paper's Interpolate; reading R20).  The MHD variables
// live at the centres of nx * ny * (nz-1) cells, the RT nodes are the cell corners: x and y are
// periodic, the corner levels below / above the box repeat the edge cell level.
// One thread owns a corner column (i, j) of a z chunk and marches up: the 4-cell horizontal sum of a
// level is formed once (fp64: exact) and used by the two corner levels that touch it, so a node
// costs 4 coalesced loads per field instead of 8.  node = (float)((h_below + h_above) / 8): the
// correctly rounded mean, bit-identical to the oracle.  Up to 3 fields per launch.
struct StaggerParams {
    int nx, ny, nz;          // RT node grid (nz = cell levels + 1)
    int nf, zchunk;
    const float* cell[3];    // [nz-1][ny][nx]
    float* node[3];          // [nz][ny][nx]
};

__global__ void __launch_bounds__(256) rts_cells_to_nodes_kernel(const StaggerParams p)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y;
    if (i >= p.nx || j >= p.ny) return;
    const int k0 = blockIdx.z * p.zchunk, k1 = min(p.nz, k0 + p.zchunk);
    const int im = (i == 0) ? p.nx - 1 : i - 1, jm = (j == 0) ? p.ny - 1 : j - 1;
    const size_t r0 = (size_t)j * p.nx, r1 = (size_t)jm * p.nx, plane = (size_t)p.nx * p.ny;
    const int ncz = p.nz - 1;
    for (int f = 0; f < p.nf; ++f) {
        const float* __restrict__ c = p.cell[f];
        float* __restrict__ n = p.node[f];
        // the four cells of a level around the corner column, as loaded (level clamped into the cell grid: the corner
        // levels below / above the box repeat the edge cell level, so k = 0 and k = nz - 1 get the same sum twice)
        auto hload = [&](int kc, float (&v)[4]) {
            const float* q = c + (size_t)min(max(kc, 0), ncz - 1) * plane;
            v[0] = __ldg(q + r0 + i); v[1] = __ldg(q + r0 + im); v[2] = __ldg(q + r1 + i); v[3] = __ldg(q + r1 + im);
        };
        auto hsum = [](const float (&v)[4]) { return ((double)v[0] + (double)v[1]) + ((double)v[2] + (double)v[3]); };
        float v0[4];
        hload(k0 - 1, v0);
        double below = hsum(v0);
        // LB levels per turn: all their loads are issued before the first store (the compiler does not move loads
        // across the stores of an unrolled loop by itself, and one level at a time is a chain of memory latencies)
        constexpr int LB = 4;
        for (int k = k0; k < k1; k += LB) {
            float v[LB][4];
#pragma unroll
            for (int u = 0; u < LB; ++u) hload(k + u, v[u]);
#pragma unroll
            for (int u = 0; u < LB; ++u) {
                if (k + u < k1) {
                    const double above = hsum(v[u]);
                    n[(size_t)(k + u) * plane + r0 + i] = (float)((below + above) * 0.125);
                    below = above;
                }
            }
        }
    }
}

// Qc(i,j,k) = mean of the 8 corner nodes of cell (i,j,k), k = 0..nz-2 (fp32; the heating goes back to
// the MHD grid).  Same marching scheme.
__global__ void __launch_bounds__(256) rts_nodes_to_cells_kernel(const float* __restrict__ qn, float* __restrict__ qc,
                                                                  int nx, int ny, int nz, int zchunk)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y;
    if (i >= nx || j >= ny) return;
    const int k0 = blockIdx.z * zchunk, k1 = min(nz - 1, k0 + zchunk);
    const int ip = (i == nx - 1) ? 0 : i + 1, jp = (j == ny - 1) ? 0 : j + 1;
    const size_t r0 = (size_t)j * nx, r1 = (size_t)jp * nx, plane = (size_t)nx * ny;
    auto hsum = [&](int k) {
        const float* q = qn + (size_t)min(k, nz - 1) * plane;
        return (__ldg(q + r0 + i) + __ldg(q + r0 + ip)) + (__ldg(q + r1 + i) + __ldg(q + r1 + ip));
    };
    if (k0 >= k1) return;
    float below = hsum(k0);
    constexpr int LB = 4;                // levels whose loads are issued before the first store (see cells -> nodes)
    for (int k = k0; k < k1; k += LB) {
        float above[LB];
#pragma unroll
        for (int u = 0; u < LB; ++u) above[u] = hsum(k + u + 1);
#pragma unroll
        for (int u = 0; u < LB; ++u) {
            if (k + u < k1) {
                qc[(size_t)(k + u) * plane + r0 + i] = 0.125f * (below + above[u]);
                below = above[u];
            }
        }
    }
}

}  // namespace rts
