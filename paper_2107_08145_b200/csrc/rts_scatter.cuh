// Scattering source function with the source update along the ray ("a
// Gauss-Seidel convergence scheme ... updating the source function for each point along the ray, and then using
// the 'new' source function to integrate the intensity at the next point along the ray.  This algorithm requires a
// combined treatment of interpolation and integration"; reading R23).  Per band (the bands of a call are
// independent problems that share every plane step and its barrier):
//     S = (1 - eps) J + eps B,   J = sum_r w_r I_r,
// the rays visited in index order, the planes of a ray along its exit-face axis in upwind order, all nodes of a plane
// at once (they read the previous plane only), one Jacobi-seam pass of the periodic faces per iteration.
//
// A first, plain kernel: fp64 throughout, one persistent cooperative grid, a grid-wide barrier after every plane
// (the update of S couples every ray to the one before it, so the 24 rays cannot run side by side as they do in
// rts_sweep_kernel).  It is launch- and barrier-bound at the sizes tested; DESIGN.md 7.5 has the numbers.
#pragma once
#include <cstdint>

namespace rts {

struct ScatRay {
    int as, dir, kdir, up;             // exit-face axis, direction along it, Dirichlet level, mu_z > 0
    int iface, jface;                  // periodic faces kept from the previous iteration
    int off[4][3];                     // the 4 stencil nodes of the upwind face (i, j, k offsets)
    double w[4];                       // their bilinear weights
    double ds, wq;                     // path length to the upwind face; quadrature weight
};

struct ScatParams {
    int nx, ny, nz, nrays, niter, gs, nb;
    const float* kaprho; const float* B; const float* eps;    // [nb][N] each
    float* kapT; float* BT; float* epsT;   // [nb][nz][nx][ny] (y fastest) copies of the three inputs, made by the kernel: the
                                           // x-march rays read them with unit stride (their planes have no x extent)
    const ScatRay* rays;
    double* I;                         // [nb][nrays][N]
    double* faceX; double* faceY;      // [nb][nz][ny], [nb][nz][nx]
    double* Sold;                      // [nb][N]
    double* S; double* J;              // [nb][N] outputs
    unsigned long long* chg;           // [niter][nb][2]: bit patterns of max |S - Sold|, max |S|
    unsigned* bar;                     // [0] arrivals (monotonic), [1] abort flag
};

// grid-wide barrier on a monotonic counter (the grid is launched cooperatively: every CTA is resident).
// Returns false if the watchdog fired: everybody leaves.  No back-off in the spin: at most a few hundred CTAs poll one
// word, and a plane step is a few microseconds.
__device__ __forceinline__ bool scat_grid_sync(unsigned* bar, unsigned& gen)
{
    __syncthreads();
    __shared__ int ok;
    if (threadIdx.x == 0) {
        ++gen;
        __threadfence();
        atomicAdd(bar, 1u);
        const unsigned need = gen * gridDim.x;
        unsigned spins = 0;
        int good = 1;
        while (true) {
            unsigned v;
            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(bar) : "memory");
            if (v >= need) break;
            if (*reinterpret_cast<volatile unsigned*>(bar + 1) != 0u) { good = 0; break; }
            if (++spins > (1u << 28)) { atomicExch(bar + 1, 1u); good = 0; break; }      // ~10 s: the watchdog
        }
        ok = good;
    }
    __syncthreads();
    return ok != 0;
}

// E = e^-dtau, psi_u, psi_p of the linear-source integration (series below 1e-3 where the closed forms cancel)
__device__ __forceinline__ void scat_psi(const double d, double& E, double& pu, double& pp)
{
    E = exp(-d);
    if (d < 1e-3) {
        pp = d * (0.5 - d * (1.0 / 6.0 - d * (1.0 / 24.0 - d * (1.0 / 120.0))));
        pu = d * (0.5 - d * (1.0 / 3.0 - d * (1.0 / 8.0 - d * (1.0 / 30.0))));
    } else {
        const double w1 = (1.0 - E) / d;
        pu = w1 - E; pp = 1.0 - w1;
    }
}

// MINB CTAs per SM: 2 (98 registers, no spills) for planes that 2 x 256 threads per SM cover with one node per thread,
// 3 (80 registers, 120 bytes of spills) for larger ones, where a second node per thread doubles the dependent chain of a
// plane step (288^3, one band: 80 -> 63 ms per iteration; 96^3: 10.5 -> 11.4 ms, hence both).  The build for large planes
// also keeps y-fastest copies of kaprho, B and eps, and stores I_r y-fastest, for the x-march rays, whose planes have no x extent: every access
// of theirs is a 32-byte sector for 4 or 8 bytes, and these three arrays are 7 of their 13 strided accesses per node
// (288^3: one band 63 -> 57 ms, four bands in one call 276 -> 206 ms; on small planes, which are latency-bound, the
// extra index arithmetic costs more than the sectors: 144^3 18.1 -> 19.7 ms, hence not there).
template <int MINB>
__global__ void __launch_bounds__(256, MINB) rts_scatter_kernel(const ScatParams p)
{
    constexpr bool UT = (MINB == 3);     // the build for large planes reads y-fastest copies of the inputs on x-march rays
    const int nx = p.nx, ny = p.ny, nz = p.nz, nb = p.nb;
    const size_t N = (size_t)nx * ny * nz, NB = N * nb;
    const size_t gtid = (size_t)blockIdx.x * blockDim.x + threadIdx.x, gsz = (size_t)gridDim.x * blockDim.x;
    unsigned gen = 0;
    const int dim[3] = {nx, ny, nz};
    const size_t fxs = (size_t)nz * ny, fys = (size_t)nz * nx;      // one band's faces

    // start: S = B, I_r = I(0) (S everywhere, 0 on the top plane of a downward ray), J = sum_r w_r I_r
    for (size_t e = gtid; e < NB; e += gsz) {
        const size_t b = e / N, n = e - b * N;
        const double bv = (double)p.B[e];
        const int k = (int)(n / ((size_t)nx * ny));
        const int jj = (int)((n / (size_t)nx) % (size_t)ny), ii = (int)(n % (size_t)nx);
        const size_t nT = ((size_t)k * nx + ii) * ny + jj;       // the node in a y-fastest array
        double j = 0.0;
        for (int r = 0; r < p.nrays; ++r) {
            const ScatRay& q = p.rays[r];
            const double i0 = (k == q.kdir && !q.up) ? 0.0 : bv;
            p.I[(b * p.nrays + r) * N + ((UT && q.as == 0) ? nT : n)] = i0;
            j += q.wq * i0;
        }
        p.S[e] = bv; p.J[e] = j;
        if (UT) { p.kapT[b * N + nT] = p.kaprho[e]; p.BT[b * N + nT] = p.B[e]; p.epsT[b * N + nT] = p.eps[e]; }
    }
    if (!scat_grid_sync(p.bar, gen)) return;

    for (int it = 0; it < p.niter; ++it) {
        for (size_t e = gtid; e < NB; e += gsz) p.Sold[e] = p.S[e];
        for (int r = 0; r < p.nrays; ++r) {
            // the ray's constants through shared memory (uniform reads), not 30 registers per thread: the large-plane build
            // spilled them (288^3: 51.5 -> 40.6 ms per iteration)
            __shared__ ScatRay qsh;
            __syncthreads();
            if (threadIdx.x < sizeof(ScatRay) / 4) reinterpret_cast<int*>(&qsh)[threadIdx.x] = reinterpret_cast<const int*>(p.rays + r)[threadIdx.x];
            __syncthreads();
            const ScatRay& q = qsh;
            // the periodic faces of the previous iteration (Jacobi seam ghosts)
            const size_t nface = (size_t)nz * (ny + nx);
            for (size_t e = gtid; e < nface * nb; e += gsz) {
                const size_t b = e / nface, f = e - b * nface;
                const double* X = p.I + (b * p.nrays + r) * N;
                const int k = (int)(f / (size_t)(ny + nx)), t = (int)(f - (size_t)k * (ny + nx));
                const bool xt = UT && (q.as == 0);               // this ray's intensity is stored y-fastest
                if (t < ny) p.faceX[b * fxs + (size_t)k * ny + t] = X[xt ? ((size_t)k * nx + q.iface) * ny + t : ((size_t)k * ny + t) * nx + q.iface];
                else p.faceY[b * fys + (size_t)k * nx + (t - ny)] = X[xt ? ((size_t)k * nx + (t - ny)) * ny + q.jface : ((size_t)k * ny + q.jface) * nx + (t - ny)];
            }
            if (!scat_grid_sync(p.bar, gen)) return;
            const int as = q.as, ua = (as == 0) ? 1 : 0, va = (as == 2) ? 1 : 2;
            const int n_u = dim[ua], n_v = dim[va], n_m = dim[as];
            const size_t npl = (size_t)n_u * n_v;
            for (int mm = 0; mm < n_m; ++mm) {
                const int pl = (q.dir > 0) ? mm : n_m - 1 - mm;
                for (size_t e = gtid; e < npl * nb; e += gsz) {
                    const size_t b = e / npl, ep = e - b * npl;
                    double* const X = p.I + (b * p.nrays + r) * N;
                    const double* const Sb = p.S + b * N;
                    // coefficient arrays: the y-fastest copies for an x-march ray
                    const bool xm = UT && (as == 0);
                    const float* const kb = (xm ? p.kapT : p.kaprho) + b * N;
                    const float* const eb = (xm ? p.epsT : p.eps) + b * N;
                    const float* const Bb = (xm ? p.BT : p.B) + b * N;
                    const double* const fX = p.faceX + b * fxs;
                    const double* const fY = p.faceY + b * fys;
                    int idx[3];
                    idx[as] = pl; idx[va] = (int)(ep / n_u); idx[ua] = (int)(ep - (size_t)idx[va] * n_u);
                    const int i = idx[0], j = idx[1], k = idx[2];
                    const size_t n = ((size_t)k * ny + j) * nx + i;
                    const size_t nc = xm ? ((size_t)k * nx + i) * ny + j : n;       // the node in the coefficient arrays and in I_r
                    // every load of the node is issued before the first use: the plane step is a chain of memory latencies,
                    // and a branch around a load (seam ghost or not; Gauss-Seidel or not) would put it behind the others
                    const size_t g = b * N + n;
                    const double Sn = Sb[n];
                    const double Xold = X[nc], Jold = p.J[g];
                    const float kn = kb[nc], epn = eb[nc], Bn = Bb[nc];
                    double Inew;
                    if (k == q.kdir) Inew = q.up ? Sn : 0.0;
                    else {
                        double xv[4], sv[4];
                        float kv[4];
#pragma unroll
                        for (int t = 0; t < 4; ++t) {
                            int iu = i + q.off[t][0], ju = j + q.off[t][1];
                            const int kq = k + q.off[t][2];
                            bool wx = false, wy = false;
                            if (iu < 0) { iu += nx; wx = true; } else if (iu >= nx) { iu -= nx; wx = true; }
                            if (ju < 0) { ju += ny; wy = true; } else if (ju >= ny) { ju -= ny; wy = true; }
                            const size_t m = ((size_t)kq * ny + ju) * nx + iu;
                            const size_t mc = xm ? ((size_t)kq * nx + iu) * ny + ju : m;   // in the coefficient arrays and in I_r
                            // a stencil node beyond a periodic seam comes from the face of the previous iteration
                            const double* const src = wx ? fX + ((size_t)kq * ny + ju) : (wy ? fY + ((size_t)kq * nx + iu) : X + mc);
                            xv[t] = *src; kv[t] = kb[mc]; sv[t] = Sb[m];
                        }
                        double Xu = 0.0, ku = 0.0, Su = 0.0;
#pragma unroll
                        for (int t = 0; t < 4; ++t) { Xu += q.w[t] * xv[t]; ku += q.w[t] * (double)kv[t]; Su += q.w[t] * sv[t]; }
                        const double dtau = 0.5 * (ku + (double)kn) * q.ds;
                        double E, pu, pp;
                        scat_psi(dtau, E, pu, pp);
                        Inew = Xu * E + pu * Su + pp * Sn;
                    }
                    if (p.gs) {
                        const double jn = Jold + q.wq * (Inew - Xold);
                        const double ep_ = (double)epn;
                        p.J[g] = jn;
                        p.S[g] = (1.0 - ep_) * jn + ep_ * (double)Bn;
                    }
                    X[nc] = Inew;
                }
                if (!scat_grid_sync(p.bar, gen)) return;
            }
        }
        if (!p.gs) {
            for (size_t e = gtid; e < NB; e += gsz) {
                const size_t b = e / N, n = e - b * N;
                const int kk = (int)(n / ((size_t)nx * ny)), jj = (int)((n / (size_t)nx) % (size_t)ny), ii = (int)(n % (size_t)nx);
                const size_t nT = ((size_t)kk * nx + ii) * ny + jj;
                double a = 0.0;
                for (int r = 0; r < p.nrays; ++r) a += p.rays[r].wq * p.I[(b * p.nrays + r) * N + ((UT && p.rays[r].as == 0) ? nT : n)];
                const double ep_ = (double)p.eps[e];
                p.J[e] = a;
                p.S[e] = (1.0 - ep_) * a + ep_ * (double)p.B[e];
            }
        }
        // change of this iteration per band (positive doubles order like their bit patterns)
        for (int b = 0; b < nb; ++b) {
            double e = 0.0, sc = 0.0;
            for (size_t n = gtid; n < N; n += gsz) { const double s = p.S[b * N + n]; e = fmax(e, fabs(s - p.Sold[b * N + n])); sc = fmax(sc, fabs(s)); }
            for (int o = 16; o > 0; o >>= 1) { e = fmax(e, __shfl_xor_sync(0xffffffffu, e, o)); sc = fmax(sc, __shfl_xor_sync(0xffffffffu, sc, o)); }
            if ((threadIdx.x & 31) == 0) {
                atomicMax(p.chg + 2 * ((size_t)it * nb + b), (unsigned long long)__double_as_longlong(e));
                atomicMax(p.chg + 2 * ((size_t)it * nb + b) + 1, (unsigned long long)__double_as_longlong(sc));
            }
        }
        if (!scat_grid_sync(p.bar, gen)) return;
    }
}

}  // namespace rts
