/*
 * rts_oracle.c -- plain fp64 CPU oracle of the RTS hot path.
 *
 * TEST INFRASTRUCTURE.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call this file.  It
 * shares no code, header, table or helper with the CUDA path under
 * paper_2107_08145_b200/csrc/ and is never used by the product path.
 *
 * What it computes (paper: arxiv 2107.08145, /root/reference/PAPER.md):
 *   PAPER.md:72  (sec. 2)   short characteristics, 24 Carlson directions, block-local
 *                           solve started from previous-iteration boundary intensities,
 *                           iterated 3-4 times
 *   PAPER.md:78-82 (sec. 2) the four RTS sub-routines Interpolate / Integrate /
 *                           Exchange / Flux
 *   PAPER.md:189 (sec. 5.1) "integrating the radiation transfer equation along a ray
 *                           using values of intensity and opacity interpolated from the
 *                           neighbouring grid cells", 3 rays per octant
 *   PAPER.md:195 (sec. 5.1) multi-band opacities; radiative heating per grid point
 *   PAPER.md:197-217 (Fig. 8) loop nest: rays x { interpol; iterate integrate; flux }
 *   PAPER.md:231 (Fig. 9)   preloaded boundary layer, each point depends on up to four
 *                           points of the previous set
 * The paper prints no formula for the scheme; every numerical choice below is the
 * reading fixed in SURVEY.md 8(c) (O-1..O-8, R1..R19) and repeated in DESIGN.md.
 *
 * The scheme is a discretisation, so the oracle is the scheme itself, step by step,
 * in the plain node order (k, j, i loops running in the ray's direction): no tiles,
 * no hyperplanes, no blocking, no fusion.
 *
 * Pins (tests/test_oracle_pins.py): exp(-tau) attenuation, linear-in-tau source,
 * optically thick limit and second moment of the ray set, isothermal exactness,
 * rotation/mirror symmetry, 1-D reduction against an independent recurrence,
 * memoised recursive evaluator on tiny grids, pass fixed point, I-form vs D-form,
 * table stage closed forms, psi check values of SURVEY 8(c) O-6; staggering (O-9):
 * constants, midpoints of linear fields, Fourier-mode attenuation cos(pi m/n),
 * edge levels, sum rule of the back-averaging; flux (O-10 / O-11): thick-limit closed form of all
 * three components, isothermal zero, mirror flip, numpy gradient, telescoping, blend weights;
 * error-controlled iteration (O-12): bit-identity with the pinned fixed-pass sweep at equal pass
 * counts, err_p = face change of consecutive fixed-pass solutions, stop rule, warm start = one
 * more pass; scattering with the source update along the ray (O-13): eps = 1 reduces to the pinned
 * fixed-pass sweeps, the converged S solves the dense linear system built from them, J bookkeeping,
 * faster than the Jacobi form, sqrt(eps) law of the isothermal semi-infinite atmosphere.
 * Parity: pinned.
 *
 * Layout: all fields [nz][ny][nx], x fastest, idx = (k*ny + j)*nx + i; z is up,
 * k = 0 is the bottom.  cgs units.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <stddef.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define SIGMA_SB 5.670374e-5
#define ORACLE_PI 3.14159265358979323846

/* ---------------------------------------------------------------------------
 * O-2  Coefficient stage (paper's interpol() minus the grid staggering,
 *      PAPER.md:79, 204).  Per node and band:
 *        x_T = (log10 T - logT_min)/(logT_max - logT_min)*(nT-1), clamped to [0,nT-1]
 *        i0 = min(floor(x_T), nT-2), t = x_T - i0;   same for P -> j0, u
 *        log10 kappa_b = bilinear(L_b; i0,t; j0,u);  kaprho_b = 10^(log10 kappa_b)*rho
 *        f_b = (1-t) f[b][i0] + t f[b][i0+1];        S_b = f_b * sigma T^4 / pi
 * O-1: inputs are the fp32 arrays, promoted to fp64 on read.
 * ------------------------------------------------------------------------- */
int oracle_coefficients(int nx, int ny, int nz, int nb, int nT, int nP,
                        double logT_min, double logT_max, double logP_min, double logP_max,
                        const float* logkappa, const float* bandfrac,
                        const float* rho, const float* T, const float* P,
                        double* kaprho, double* S)
{
    if (nx < 1 || ny < 1 || nz < 1 || nb < 1 || nT < 2 || nP < 2) return -1;
    const size_t N = (size_t)nx * ny * nz;
    long n;
#pragma omp parallel for schedule(static)
    for (n = 0; n < (long)N; ++n) {
        double xT = (log10((double)T[n]) - logT_min) / (logT_max - logT_min) * (nT - 1);
        double xP = (log10((double)P[n]) - logP_min) / (logP_max - logP_min) * (nP - 1);
        if (xT < 0.0) xT = 0.0;
        if (xT > nT - 1) xT = nT - 1;
        if (xP < 0.0) xP = 0.0;
        if (xP > nP - 1) xP = nP - 1;
        int i0 = (int)floor(xT); if (i0 > nT - 2) i0 = nT - 2;
        int j0 = (int)floor(xP); if (j0 > nP - 2) j0 = nP - 2;
        double t = xT - i0, u = xP - j0;
        double Tn = (double)T[n];
        double planck = SIGMA_SB * Tn * Tn * Tn * Tn / ORACLE_PI;
        for (int b = 0; b < nb; ++b) {
            const float* L = logkappa + (size_t)b * nT * nP;
            double lk = (1.0 - t) * (1.0 - u) * (double)L[(size_t)i0 * nP + j0]
                      + t * (1.0 - u) * (double)L[(size_t)(i0 + 1) * nP + j0]
                      + (1.0 - t) * u * (double)L[(size_t)i0 * nP + j0 + 1]
                      + t * u * (double)L[(size_t)(i0 + 1) * nP + j0 + 1];
            double fb = (1.0 - t) * (double)bandfrac[(size_t)b * nT + i0]
                      + t * (double)bandfrac[(size_t)b * nT + i0 + 1];
            kaprho[(size_t)b * N + n] = pow(10.0, lk) * (double)rho[n];
            S[(size_t)b * N + n] = fb * planck;
        }
    }
    return 0;
}

/* ---------------------------------------------------------------------------
 * O-3  Ray geometry.  t_a = h_a/|mu_a|; ds = min_a t_a; entry-face axis a* = argmin
 *      (ties: prefer z, then y, then x); for the two other axes f_c = ds*|mu_c|/h_c.
 *      sgn[a] = +1 if mu_a >= 0 else -1.
 * ------------------------------------------------------------------------- */
int oracle_ray_geometry(double dx, double dy, double dz, const double* mu,
                        int* axis, int* sgn, double* ds, double* f)
{
    const double h[3] = {dx, dy, dz};
    double t[3];
    for (int a = 0; a < 3; ++a) {
        sgn[a] = (mu[a] >= 0.0) ? 1 : -1;
        t[a] = (mu[a] != 0.0) ? h[a] / fabs(mu[a]) : HUGE_VAL;
    }
    if (mu[2] == 0.0) return -1;           /* horizontal rays have no inflow boundary here */
    int as = 2;                            /* prefer z, then y, then x on ties */
    if (t[1] < t[as]) as = 1;
    if (t[0] < t[as]) as = 0;
    *axis = as;
    *ds = t[as];
    for (int a = 0; a < 3; ++a) f[a] = (a == as) ? 1.0 : (*ds) * fabs(mu[a]) / h[a];
    return 0;
}

/* O-6 weights of the linear-source-function integration over dtau.
 *   E = exp(-dtau); w1 = (1-E)/dtau; psi_u = w1 - E; psi_p = 1 - w1.
 *   Series below dtau < 1e-3 (truncation < 2e-18). */
void oracle_psi(double dtau, double* E, double* psi_u, double* psi_p)
{
    if (dtau < 1e-3) {
        double d = dtau;
        *E = exp(-d);
        *psi_p = d / 2.0 - d * d / 6.0 + d * d * d / 24.0 - d * d * d * d / 120.0;
        *psi_u = d / 2.0 - d * d / 3.0 + d * d * d / 8.0 - d * d * d * d / 30.0;
    } else {
        double e = exp(-dtau);
        double w1 = (1.0 - e) / dtau;
        *E = e;
        *psi_u = w1 - e;
        *psi_p = 1.0 - w1;
    }
}

/* One pass of O-5 in place: X holds pass p-1 on entry and pass p on exit; faceX / faceY are the
 * faces i = iface and j = jface of pass p-1 (the only values of pass p-1 that are read). */
static void sweep_one_pass(int nx, int ny, int nz, int sx, int sy, int sz, int kdir,
                           int off[4][3], const double* w, double ds,
                           const double* kaprho, const double* S, int form,
                           const double* faceX, const double* faceY, double* X)
{
    for (int kk = 0; kk < nz; ++kk) {
        int k = (sz > 0) ? kk : nz - 1 - kk;
        if (k == kdir) continue;                        /* Dirichlet plane: not updated */
        for (int jj = 0; jj < ny; ++jj) {
            int j = (sy > 0) ? jj : ny - 1 - jj;
            for (int ii = 0; ii < nx; ++ii) {
                int i = (sx > 0) ? ii : nx - 1 - ii;
                size_t n = ((size_t)k * ny + j) * nx + i;
                double Xu = 0.0, ku = 0.0, Su = 0.0;
                for (int q = 0; q < 4; ++q) {
                    int iu = i + off[q][0], ju = j + off[q][1], kq = k + off[q][2];
                    int wrapx = 0, wrapy = 0;
                    if (iu < 0) { iu += nx; wrapx = 1; } else if (iu >= nx) { iu -= nx; wrapx = 1; }
                    if (ju < 0) { ju += ny; wrapy = 1; } else if (ju >= ny) { ju -= ny; wrapy = 1; }
                    /* kq stays inside [0,nz): the Dirichlet plane is never updated */
                    size_t m = ((size_t)kq * ny + ju) * nx + iu;
                    double xv;
                    if (wrapx) xv = faceX[(size_t)kq * ny + ju];       /* iu == iface */
                    else if (wrapy) xv = faceY[(size_t)kq * nx + iu];  /* ju == jface */
                    else xv = X[m];
                    Xu += w[q] * xv;
                    ku += w[q] * kaprho[m];
                    Su += w[q] * S[m];
                }
                double dtau = 0.5 * (ku + kaprho[n]) * ds;
                double E, pu, pp;
                oracle_psi(dtau, &E, &pu, &pp);
                if (!form) {
                    X[n] = Xu * E + pu * Su + pp * S[n];
                } else {
                    /* D_p = D_u E - (S_p - S_u)(1-E)/dtau ; (1-E)/dtau = E + psi_u */
                    X[n] = Xu * E - (S[n] - Su) * (E + pu);
                }
            }
        }
    }
}

/* ---------------------------------------------------------------------------
 * O-4..O-6  Formal solution for ONE band and ONE ray, all passes.
 *
 *  kaprho, S : nodal fields of this band [nz][ny][nx] (fp64)
 *  mu        : direction of photon travel
 *  I_inflow  : NULL -> the paper's boundary values (bottom I = S for mu_z > 0, top
 *              I = 0 for mu_z < 0; O-4); else [ny][nx] incoming intensity placed on the
 *              Dirichlet node plane (test hook for the exp(-tau) pin)
 *  form      : 0 = carry the intensity I (the scheme as stated);
 *              1 = carry the departure D = I - S (algebraically identical: S_u is the
 *                  bilinear interpolant of nodal S); used only to pin the conditioning
 *  I         : out, I^(P) at every node [nz][ny][nx]
 *
 *  Passes (O-5): I^(0) = Dirichlet value on the Dirichlet plane, S elsewhere.  In pass p
 *  every non-Dirichlet node is updated once in the plain upwind order.  A stencil node
 *  whose x or y index wraps takes its intensity from I^(p-1) (Jacobi ghosts); stencil
 *  nodes that do not wrap use I^(p).  Only the faces i = (sx>0 ? nx-1 : 0) and
 *  j = (sy>0 ? ny-1 : 0) of I^(p-1) are ever read, so only those are kept.
 * ------------------------------------------------------------------------- */
int oracle_sweep_ray(int nx, int ny, int nz, double dx, double dy, double dz,
                     const double* mu, int npasses,
                     const double* kaprho, const double* S,
                     const double* I_inflow, int form, double* I)
{
    int as, sg[3];
    double ds, f[3];
    if (nx < 1 || ny < 1 || nz < 2 || npasses < 1) return -1;
    if (oracle_ray_geometry(dx, dy, dz, mu, &as, sg, &ds, f) != 0) return -1;
    const int sx = sg[0], sy = sg[1], sz = sg[2];
    const size_t N = (size_t)nx * ny * nz;
    const int kdir = (sz > 0) ? 0 : nz - 1;      /* Dirichlet node plane (O-4) */

    /* the two transverse axes c, d of the entry face and the 4 stencil offsets/weights */
    int c = (as == 0) ? 1 : 0;
    int d = (as == 2) ? 1 : 2;
    int off[4][3];
    double w[4];
    for (int ec = 0; ec < 2; ++ec)
        for (int ed = 0; ed < 2; ++ed) {
            int q = ec * 2 + ed;
            off[q][0] = off[q][1] = off[q][2] = 0;
            off[q][as] = -sg[as];
            off[q][c] = -ec * sg[c];
            off[q][d] = -ed * sg[d];
            w[q] = (ec ? f[c] : 1.0 - f[c]) * (ed ? f[d] : 1.0 - f[d]);
        }

    /* work array holds the carried quantity X = I (form 0) or D = I - S (form 1) */
    double* X = I;
    double* faceX = (double*)malloc(sizeof(double) * (size_t)nz * ny);  /* X^(p-1)(i_face, j, k) */
    double* faceY = (double*)malloc(sizeof(double) * (size_t)nz * nx);  /* X^(p-1)(i, j_face, k) */
    if (!faceX || !faceY) { free(faceX); free(faceY); return -2; }
    const int iface = (sx > 0) ? nx - 1 : 0;
    const int jface = (sy > 0) ? ny - 1 : 0;

    /* I^(0) */
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                size_t n = ((size_t)k * ny + j) * nx + i;
                double I0;
                if (k == kdir) {
                    if (I_inflow) I0 = I_inflow[(size_t)j * nx + i];
                    else I0 = (sz > 0) ? S[n] : 0.0;
                } else I0 = S[n];
                X[n] = form ? I0 - S[n] : I0;
            }

    for (int p = 1; p <= npasses; ++p) {
        /* keep the two faces of pass p-1 */
        for (int k = 0; k < nz; ++k) {
            for (int j = 0; j < ny; ++j) faceX[(size_t)k * ny + j] = X[((size_t)k * ny + j) * nx + iface];
            for (int i = 0; i < nx; ++i) faceY[(size_t)k * nx + i] = X[((size_t)k * ny + jface) * nx + i];
        }
        sweep_one_pass(nx, ny, nz, sx, sy, sz, kdir, off, w, ds, kaprho, S, form, faceX, faceY, X);
    }
    if (form) for (size_t n = 0; n < N; ++n) I[n] = X[n] + S[n];
    free(faceX); free(faceY);
    return 0;
}

/* ---------------------------------------------------------------------------
 * O-12  Error-controlled iteration and warm start (Fig. 8
 *       "while(g_maxerr > THRESHOLD) { readbuf(); integrate(); writebuf(); exchange(); err = error();
 *       MPI_Allreduce(&err, &g_maxerr); }", "iterates the intensities at the boundaries
 *       ... until the errors are within a prescribed tolerance"; reading R22).
 *   The boundary intensities of the periodic box are the two faces O-5 keeps: i = iface (all j, k)
 *   and j = jface (all i, k).  After pass p
 *       err_p = max over both faces |I^(p) - I^(p-1)|,   scale_p = max over both faces |I^(p)|,
 *   and the iteration stops at the first p with err_p <= tol * scale_p, or at p = max_passes.
 *   Warm start: the faces of I^(0) are given (the converged faces of an earlier solve) instead of
 *   taken from I^(0) = S; no other value of I^(0) is ever read.
 *
 *  State of one (band, ray) problem between passes: X (the whole field) and its two faces.
 * ------------------------------------------------------------------------- */
typedef struct {
    int as, sx, sy, sz, kdir, iface, jface;
    int off[4][3];
    double w[4], ds;
} ray_setup;

static int ray_setup_init(int nx, int ny, int nz, double dx, double dy, double dz, const double* mu, ray_setup* r)
{
    int sg[3];
    double f[3];
    if (oracle_ray_geometry(dx, dy, dz, mu, &r->as, sg, &r->ds, f) != 0) return -1;
    r->sx = sg[0]; r->sy = sg[1]; r->sz = sg[2];
    r->kdir = (r->sz > 0) ? 0 : nz - 1;
    const int as = r->as, c = (as == 0) ? 1 : 0, d = (as == 2) ? 1 : 2;
    for (int ec = 0; ec < 2; ++ec)
        for (int ed = 0; ed < 2; ++ed) {
            int q = ec * 2 + ed;
            r->off[q][0] = r->off[q][1] = r->off[q][2] = 0;
            r->off[q][as] = -sg[as];
            r->off[q][c] = -ec * sg[c];
            r->off[q][d] = -ed * sg[d];
            r->w[q] = (ec ? f[c] : 1.0 - f[c]) * (ed ? f[d] : 1.0 - f[d]);
        }
    r->iface = (r->sx > 0) ? nx - 1 : 0;
    r->jface = (r->sy > 0) ? ny - 1 : 0;
    return 0;
}

/* I^(0) of O-5 into X; the faces of I^(0) into faceX / faceY (or the warm faces, if given) */
static void tol_init(int nx, int ny, int nz, const ray_setup* r, const double* S,
                     const double* warmX, const double* warmY, double* X, double* faceX, double* faceY)
{
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                size_t n = ((size_t)k * ny + j) * nx + i;
                X[n] = (k == r->kdir) ? ((r->sz > 0) ? S[n] : 0.0) : S[n];
            }
    for (int k = 0; k < nz; ++k) {
        for (int j = 0; j < ny; ++j)
            faceX[(size_t)k * ny + j] = warmX ? warmX[(size_t)k * ny + j] : X[((size_t)k * ny + j) * nx + r->iface];
        for (int i = 0; i < nx; ++i)
            faceY[(size_t)k * nx + i] = warmY ? warmY[(size_t)k * nx + i] : X[((size_t)k * ny + r->jface) * nx + i];
    }
}

/* one pass + error(): faces hold pass p-1 on entry and pass p on exit */
static void tol_pass(int nx, int ny, int nz, ray_setup* r, const double* kaprho, const double* S,
                     double* X, double* faceX, double* faceY, double* err, double* scale)
{
    sweep_one_pass(nx, ny, nz, r->sx, r->sy, r->sz, r->kdir, r->off, r->w, r->ds, kaprho, S, 0, faceX, faceY, X);
    double e = 0.0, sc = 0.0;
    for (int k = 0; k < nz; ++k) {
        for (int j = 0; j < ny; ++j) {
            const double v = X[((size_t)k * ny + j) * nx + r->iface], o = faceX[(size_t)k * ny + j];
            if (fabs(v - o) > e) e = fabs(v - o);
            if (fabs(v) > sc) sc = fabs(v);
            faceX[(size_t)k * ny + j] = v;
        }
        for (int i = 0; i < nx; ++i) {
            const double v = X[((size_t)k * ny + r->jface) * nx + i], o = faceY[(size_t)k * nx + i];
            if (fabs(v - o) > e) e = fabs(v - o);
            if (fabs(v) > sc) sc = fabs(v);
            faceY[(size_t)k * nx + i] = v;
        }
    }
    *err = e; *scale = sc;
}

/* ONE band and ONE ray, iterated to the tolerance.  warmX [nz][ny] / warmY [nz][nx]: faces of I^(0) or NULL.
 * Outputs: I [nz][ny][nx]; faceX_out / faceY_out (may be NULL): the faces of the final pass; relerr
 * [max_passes]: err_p / scale_p of every pass run; *passes_used. */
int oracle_sweep_ray_tol(int nx, int ny, int nz, double dx, double dy, double dz,
                         const double* mu, double tol, int max_passes,
                         const double* kaprho, const double* S,
                         const double* warmX, const double* warmY,
                         double* I, double* faceX_out, double* faceY_out, double* relerr, int* passes_used)
{
    ray_setup r;
    if (nx < 1 || ny < 1 || nz < 2 || max_passes < 1 || !passes_used) return -1;
    if (ray_setup_init(nx, ny, nz, dx, dy, dz, mu, &r) != 0) return -1;
    double* faceX = (double*)malloc(sizeof(double) * (size_t)nz * ny);
    double* faceY = (double*)malloc(sizeof(double) * (size_t)nz * nx);
    if (!faceX || !faceY) { free(faceX); free(faceY); return -2; }
    tol_init(nx, ny, nz, &r, S, warmX, warmY, I, faceX, faceY);
    int p = 0;
    while (p < max_passes) {
        double e, sc;
        tol_pass(nx, ny, nz, &r, kaprho, S, I, faceX, faceY, &e, &sc);
        if (relerr) relerr[p] = (sc > 0.0) ? e / sc : 0.0;
        ++p;
        if (e <= tol * sc) break;
    }
    *passes_used = p;
    if (faceX_out) memcpy(faceX_out, faceX, sizeof(double) * (size_t)nz * ny);
    if (faceY_out) memcpy(faceY_out, faceY, sizeof(double) * (size_t)nz * nx);
    free(faceX); free(faceY);
    return 0;
}

/* All bands and rays, iterated to the tolerance; J, Q and I_top as in O-7.
 *   mode 0: every (band, ray) problem stops on its own error (Fig. 8 read literally: the while loop
 *           is inside the ray loop);
 *   mode 1: all problems iterate together until the largest err_p / scale_p of any of them is <= tol
 *           (one pass count for the whole solve).
 *   faces: NULL, or in/out [nb*nrays][nz*ny + nz*nx]: on entry (if warm != 0) the faces of I^(0) of
 *   every problem, on exit the faces of its final pass.  passes_used [nb*nrays];  relerr (may be NULL)
 *   [max_passes]: mode 1 only, the largest err_p / scale_p of every pass run. */
int oracle_solve_tol(int nx, int ny, int nz, double dx, double dy, double dz,
                     int nb, int nT, int nP,
                     double logT_min, double logT_max, double logP_min, double logP_max,
                     const float* logkappa, const float* bandfrac,
                     double tol, int max_passes, int mode, int warm,
                     int nrays, const double* mu, const double* wq,
                     const float* rho, const float* T, const float* P,
                     double* Q, double* Itop, double* faces, int* passes_used, double* relerr, int nthreads)
{
    if (nx < 1 || ny < 1 || nz < 2 || nb < 1 || nrays < 1 || max_passes < 1 || !passes_used) return -1;
    if (warm && !faces) return -1;
    const size_t N = (size_t)nx * ny * nz, nfx = (size_t)nz * ny, nfy = (size_t)nz * nx, nf = nfx + nfy;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#else
    (void)nthreads;
#endif
    const int ntask = nb * nrays;
    double* kaprho = (double*)malloc(sizeof(double) * N * nb);
    double* S = (double*)malloc(sizeof(double) * N * nb);
    double* X = (double*)malloc(sizeof(double) * N * (size_t)ntask);      /* every problem's field */
    double* fc = (double*)malloc(sizeof(double) * nf * (size_t)ntask);    /* ... and faces */
    double* te = (double*)malloc(sizeof(double) * 2 * (size_t)ntask);
    ray_setup* rs = (ray_setup*)malloc(sizeof(ray_setup) * (size_t)nrays);
    int* done = (int*)calloc((size_t)ntask, sizeof(int));
    if (!kaprho || !S || !X || !fc || !te || !rs || !done) { free(kaprho); free(S); free(X); free(fc); free(te); free(rs); free(done); return -2; }
    int rc = oracle_coefficients(nx, ny, nz, nb, nT, nP, logT_min, logT_max, logP_min, logP_max,
                                 logkappa, bandfrac, rho, T, P, kaprho, S);
    for (int r = 0; r < nrays && rc == 0; ++r) rc = ray_setup_init(nx, ny, nz, dx, dy, dz, mu + 3 * r, &rs[r]);
    if (rc == 0) {
        int t;
#pragma omp parallel for schedule(static, 1)
        for (t = 0; t < ntask; ++t) {
            const int b = t / nrays, r = t % nrays;
            const double* wf = warm ? faces + (size_t)t * nf : NULL;
            tol_init(nx, ny, nz, &rs[r], S + (size_t)b * N, wf, wf ? wf + nfx : NULL,
                     X + (size_t)t * N, fc + (size_t)t * nf, fc + (size_t)t * nf + nfx);
            passes_used[t] = 0;
        }
        for (int p = 0; p < max_passes; ++p) {
            int active = 0;
#pragma omp parallel for schedule(static, 1) reduction(+ : active)
            for (t = 0; t < ntask; ++t) {
                if (done[t]) continue;
                const int b = t / nrays, r = t % nrays;
                ray_setup rr = rs[r];
                tol_pass(nx, ny, nz, &rr, kaprho + (size_t)b * N, S + (size_t)b * N,
                         X + (size_t)t * N, fc + (size_t)t * nf, fc + (size_t)t * nf + nfx, &te[2 * t], &te[2 * t + 1]);
                passes_used[t] = p + 1;
                ++active;
            }
            if (!active) break;
            double worst = 0.0;
            for (t = 0; t < ntask; ++t) {
                if (done[t]) continue;
                const double rel = (te[2 * t + 1] > 0.0) ? te[2 * t] / te[2 * t + 1] : 0.0;
                if (rel > worst) worst = rel;
                if (mode == 0 && te[2 * t] <= tol * te[2 * t + 1]) done[t] = 1;
            }
            if (mode == 1) {
                if (relerr) relerr[p] = worst;
                if (worst <= tol) break;
            }
        }
        /* J, Q, I_top in (band, ray) order at every node, as in O-7 */
        int nup = 0;
        for (int r = 0; r < nrays; ++r) nup += (mu[3 * r + 2] > 0.0);
        long n;
#pragma omp parallel for schedule(static)
        for (n = 0; n < (long)N; ++n) {
            double q = 0.0;
            for (int b = 0; b < nb; ++b) {
                double J = 0.0;
                for (int r = 0; r < nrays; ++r) J += wq[r] * X[((size_t)b * nrays + r) * N + n];
                q += 4.0 * ORACLE_PI * kaprho[(size_t)b * N + n] * (J - S[(size_t)b * N + n]);
            }
            Q[n] = q;
        }
        if (Itop) {
            int u = 0;
            for (int r = 0; r < nrays; ++r) {
                if (!(mu[3 * r + 2] > 0.0)) continue;
                for (int b = 0; b < nb; ++b)
                    memcpy(Itop + ((size_t)b * nup + u) * ny * nx,
                           X + ((size_t)b * nrays + r) * N + (size_t)(nz - 1) * ny * nx, sizeof(double) * ny * nx);
                ++u;
            }
        }
        if (faces) memcpy(faces, fc, sizeof(double) * nf * (size_t)ntask);
    }
    free(kaprho); free(S); free(X); free(fc); free(te); free(rs); free(done);
    return rc;
}

/* ---------------------------------------------------------------------------
 * O-7  Full solve: all bands, all rays, J, Q and I_top (+ O-10 radiative flux).
 *   J_b = sum_r w_r I_{b,r}^(P);  Q = 4 pi sum_b kaprho_b (J_b - S_b) at every node;
 *   Itop[b][u][j][i] = I_{b,r}^(P)(i,j,nz-1) for the u-th ray with mu_z > 0 (in ray order).
 *   O-10 (paper's Flux, "From the specific intensity calculate the
 *   average intensity and radiative fluxes"; reading R21):
 *     F_a = 4 pi sum_b sum_r w_r Omega_{r,a} I_{b,r}^(P),  Omega_r = mu_r / |mu_r|,  a = x, y, z.
 *   Optional outputs (may be NULL): Jout [nb][N], Fout [3][N].
 *   nthreads <= 0: all OpenMP threads.
 *   The (band, ray) sweeps are independent; they run in batches of one sweep per thread and
 *   each batch is added to J (and F) in (band, ray) order by a loop over the nodes, so the
 *   sums are formed in the same order for any thread count.
 * ------------------------------------------------------------------------- */
int oracle_solve(int nx, int ny, int nz, double dx, double dy, double dz,
                 int nb, int nT, int nP,
                 double logT_min, double logT_max, double logP_min, double logP_max,
                 const float* logkappa, const float* bandfrac,
                 int npasses, int nrays, const double* mu, const double* wq,
                 const float* rho, const float* T, const float* P,
                 double* Q, double* Itop, double* Jout, double* Fout, int nthreads)
{
    if (nx < 1 || ny < 1 || nz < 2 || nb < 1 || nrays < 1) return -1;
    const size_t N = (size_t)nx * ny * nz;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
    const int nt = omp_get_max_threads();
#else
    (void)nthreads;
    const int nt = 1;
#endif
    const int ntask = nb * nrays;
    const int batch = nt < ntask ? nt : ntask;
    double* kaprho = (double*)malloc(sizeof(double) * N * nb);
    double* S = (double*)malloc(sizeof(double) * N * nb);
    double* J = (double*)calloc(N * nb, sizeof(double));
    double* Ibuf = (double*)malloc(sizeof(double) * N * (size_t)batch);
    int* upidx = (int*)malloc(sizeof(int) * nrays);
    int* err = (int*)calloc((size_t)batch, sizeof(int));
    if (!kaprho || !S || !J || !upidx || !Ibuf || !err) { free(kaprho); free(S); free(J); free(upidx); free(Ibuf); free(err); return -2; }
    int rc = oracle_coefficients(nx, ny, nz, nb, nT, nP, logT_min, logT_max, logP_min, logP_max,
                                 logkappa, bandfrac, rho, T, P, kaprho, S);
    int nup = 0;
    for (int r = 0; r < nrays; ++r) upidx[r] = (mu[3 * r + 2] > 0.0) ? nup++ : -1;
    if (Fout) memset(Fout, 0, sizeof(double) * 3 * N);

    int fail = rc;
    for (int t0 = 0; t0 < ntask && fail == 0; t0 += batch) {
        const int nb_ = (ntask - t0 < batch) ? ntask - t0 : batch;
        int q;
#pragma omp parallel for schedule(static, 1)
        for (q = 0; q < nb_; ++q) {
            const int task = t0 + q, b = task / nrays, r = task % nrays;
            double* I = Ibuf + (size_t)q * N;
            err[q] = oracle_sweep_ray(nx, ny, nz, dx, dy, dz, mu + 3 * r, npasses,
                                      kaprho + (size_t)b * N, S + (size_t)b * N, NULL, 0, I);
            if (err[q] == 0 && Itop && upidx[r] >= 0) {
                double* dst = Itop + ((size_t)b * nup + upidx[r]) * ny * nx;
                memcpy(dst, I + (size_t)(nz - 1) * ny * nx, sizeof(double) * ny * nx);
            }
        }
        for (q = 0; q < nb_; ++q) if (err[q] != 0) fail = err[q];
        if (fail != 0) break;
        /* J_b += w_r I_r and F += 4 pi w_r Omega_r I_r, in (band, ray) order at every node */
        long n;
#pragma omp parallel for schedule(static)
        for (n = 0; n < (long)N; ++n) {
            for (int qq = 0; qq < nb_; ++qq) {
                const int task = t0 + qq, b = task / nrays, r = task % nrays;
                const double Iv = Ibuf[(size_t)qq * N + n];
                J[(size_t)b * N + n] += wq[r] * Iv;
                if (Fout) {
                    const double* m = mu + 3 * r;
                    const double nrm = sqrt(m[0] * m[0] + m[1] * m[1] + m[2] * m[2]);
                    for (int a = 0; a < 3; ++a) Fout[(size_t)a * N + n] += 4.0 * ORACLE_PI * wq[r] * (m[a] / nrm) * Iv;
                }
            }
        }
    }
    if (fail == 0) {
        long n;
#pragma omp parallel for schedule(static)
        for (n = 0; n < (long)N; ++n) {
            double q = 0.0;
            for (int b = 0; b < nb; ++b)
                q += 4.0 * ORACLE_PI * kaprho[(size_t)b * N + n] * (J[(size_t)b * N + n] - S[(size_t)b * N + n]);
            Q[n] = q;
        }
        if (Jout) memcpy(Jout, J, sizeof(double) * N * nb);
    }
    free(kaprho); free(S); free(J); free(upidx); free(Ibuf); free(err);
    return fail;
}

/* ---------------------------------------------------------------------------
 * O-13  Scattering source function with the source update along the ray (
 *       PAPER.md:261 "it is preferable to use a Gauss-Seidel convergence scheme.  As the intensity is
 *       integrated along the ray, this scheme will require updating the source function for each point
 *       along the ray, and then using the 'new' source function to integrate the intensity at the next
 *       point along the ray.  This algorithm requires a combined treatment of interpolation and
 *       integration."; reading R23).  ONE band:
 *           S = (1 - eps) J + eps B,    J = sum_r w_r I_r,
 *       eps: photon destruction probability per node (0 < eps <= 1; eps = 1 is the LTE path), B: the
 *       thermal source of stage A, I_r: the short-characteristic solution of O-4..O-6 for the current S.
 *       Start: S = B, I_r = I^(0) of O-5 for S = B, J = sum_r w_r I_r.
 *       One iteration visits the rays in index order.  For ray r the faces of I_r of the previous
 *       iteration are kept (Jacobi ghosts of O-5: one pass per iteration), then the planes along the
 *       ray's exit-face axis are visited in upwind order; every node n of a plane
 *           I_new = I_u E + psi_u S_u + psi_p S[n]        (S_u: bilinear over the previous plane, S as it is NOW)
 *                   (Dirichlet node, O-4: I_new = S[n] for an upward ray, 0 for a downward one)
 *         gs = 1 (the paper's scheme):  J[n] += w_r (I_new - I_r[n]);  I_r[n] = I_new;
 *                                       S[n] = (1 - eps[n]) J[n] + eps[n] B[n]
 *         gs = 0 (Jacobi / Lambda iteration, the comparison):  I_r[n] = I_new only; after the last ray
 *                                       J = sum_r w_r I_r and S = (1 - eps) J + eps B at every node.
 *       The nodes of one plane do not read each other (all stencil nodes lie in the previous plane), so the
 *       order inside a plane is immaterial.  change[it] = max_n |S_new - S_old| / max_n |S_new| of iteration it.
 *  Outputs: S, J [N]; Iall (may be NULL) [nrays][N]; change [niter].
 * ------------------------------------------------------------------------- */
int oracle_scatter_solve(int nx, int ny, int nz, double dx, double dy, double dz,
                         int nrays, const double* mu, const double* wq,
                         const double* kaprho, const double* B, const double* eps,
                         int niter, int gs, double* S, double* J, double* Iall, double* change)
{
    if (nx < 1 || ny < 1 || nz < 2 || nrays < 1 || niter < 0) return -1;
    const size_t N = (size_t)nx * ny * nz;
    double* I = Iall ? Iall : (double*)malloc(sizeof(double) * N * (size_t)nrays);
    double* faceX = (double*)malloc(sizeof(double) * (size_t)nz * ny);
    double* faceY = (double*)malloc(sizeof(double) * (size_t)nz * nx);
    double* Sold = (double*)malloc(sizeof(double) * N);
    ray_setup* rs = (ray_setup*)malloc(sizeof(ray_setup) * (size_t)nrays);
    if (!I || !faceX || !faceY || !Sold || !rs) { if (!Iall) free(I); free(faceX); free(faceY); free(Sold); free(rs); return -2; }
    int rc = 0;
    for (int r = 0; r < nrays && rc == 0; ++r) rc = ray_setup_init(nx, ny, nz, dx, dy, dz, mu + 3 * r, &rs[r]);
    if (rc == 0) {
        for (size_t n = 0; n < N; ++n) { S[n] = B[n]; J[n] = 0.0; }
        for (int r = 0; r < nrays; ++r)
            for (int k = 0; k < nz; ++k)
                for (size_t h = 0; h < (size_t)ny * nx; ++h) {
                    const size_t n = (size_t)k * ny * nx + h;
                    const double I0 = (k == rs[r].kdir && rs[r].sz < 0) ? 0.0 : S[n];
                    I[(size_t)r * N + n] = I0;
                    J[n] += wq[r] * I0;
                }
        for (int it = 0; it < niter; ++it) {
            memcpy(Sold, S, sizeof(double) * N);
            for (int r = 0; r < nrays; ++r) {
                const ray_setup* q = &rs[r];
                double* X = I + (size_t)r * N;
                for (int k = 0; k < nz; ++k) {
                    for (int j = 0; j < ny; ++j) faceX[(size_t)k * ny + j] = X[((size_t)k * ny + j) * nx + q->iface];
                    for (int i = 0; i < nx; ++i) faceY[(size_t)k * nx + i] = X[((size_t)k * ny + q->jface) * nx + i];
                }
                /* planes along the exit-face axis `as`, upwind first; (c, d) the two other axes */
                const int as = q->as, c = (as == 0) ? 1 : 0, d = (as == 2) ? 1 : 2;
                const int dim[3] = {nx, ny, nz}, sg[3] = {q->sx, q->sy, q->sz};
                for (int mm = 0; mm < dim[as]; ++mm)
                    for (int dd = 0; dd < dim[d]; ++dd)
                        for (int cc = 0; cc < dim[c]; ++cc) {
                            int idx[3];
                            idx[as] = (sg[as] > 0) ? mm : dim[as] - 1 - mm;
                            idx[c] = cc; idx[d] = dd;
                            const int i = idx[0], j = idx[1], k = idx[2];
                            const size_t n = ((size_t)k * ny + j) * nx + i;
                            double Inew;
                            if (k == q->kdir) Inew = (q->sz > 0) ? S[n] : 0.0;
                            else {
                                double Xu = 0.0, ku = 0.0, Su = 0.0;
                                for (int t = 0; t < 4; ++t) {
                                    int iu = i + q->off[t][0], ju = j + q->off[t][1], kq = k + q->off[t][2];
                                    int wrapx = 0, wrapy = 0;
                                    if (iu < 0) { iu += nx; wrapx = 1; } else if (iu >= nx) { iu -= nx; wrapx = 1; }
                                    if (ju < 0) { ju += ny; wrapy = 1; } else if (ju >= ny) { ju -= ny; wrapy = 1; }
                                    const size_t m = ((size_t)kq * ny + ju) * nx + iu;
                                    double xv;
                                    if (wrapx) xv = faceX[(size_t)kq * ny + ju];
                                    else if (wrapy) xv = faceY[(size_t)kq * nx + iu];
                                    else xv = X[m];
                                    Xu += q->w[t] * xv;
                                    ku += q->w[t] * kaprho[m];
                                    Su += q->w[t] * S[m];
                                }
                                const double dtau = 0.5 * (ku + kaprho[n]) * q->ds;
                                double E, pu, pp;
                                oracle_psi(dtau, &E, &pu, &pp);
                                Inew = Xu * E + pu * Su + pp * S[n];
                            }
                            if (gs) {
                                J[n] += wq[r] * (Inew - X[n]);
                                S[n] = (1.0 - eps[n]) * J[n] + eps[n] * B[n];
                            }
                            X[n] = Inew;
                        }
            }
            if (!gs)
                for (size_t n = 0; n < N; ++n) {
                    double a = 0.0;
                    for (int r = 0; r < nrays; ++r) a += wq[r] * I[(size_t)r * N + n];
                    J[n] = a;
                    S[n] = (1.0 - eps[n]) * a + eps[n] * B[n];
                }
            double e = 0.0, sc = 0.0;
            for (size_t n = 0; n < N; ++n) {
                if (fabs(S[n] - Sold[n]) > e) e = fabs(S[n] - Sold[n]);
                if (fabs(S[n]) > sc) sc = fabs(S[n]);
            }
            if (change) change[it] = (sc > 0.0) ? e / sc : 0.0;
        }
    }
    if (!Iall) free(I);
    free(faceX); free(faceY); free(Sold); free(rs);
    return rc;
}

/* ---------------------------------------------------------------------------
 * O-11  Flux-divergence heating and its blend with the J - S form (
 *       DESIGN.md reading R21).  On the node grid:
 *         Qdiv = -(dFx/dx + dFy/dy + dFz/dz),
 *       central differences, periodic in x and y; on the bottom / top node plane the z
 *       derivative is the one-sided difference over one spacing.
 *         Qblend = w Q_J + (1 - w) Qdiv,   w(k) = exp(-taubar(k) / tau0),
 *       taubar(k) = sum_{k' >= k} <kaprho_0>(k') dz: the horizontally averaged optical depth of
 *       band 0 from the top down to (and including) level k.  kaprho0: [N] band-0 kaprho.
 *       Qdiv / Qblend may be NULL.
 * ------------------------------------------------------------------------- */
int oracle_flux_heating(int nx, int ny, int nz, double dx, double dy, double dz,
                        const double* F, const double* QJ, const double* kaprho0, double tau0,
                        double* Qdiv, double* Qblend)
{
    if (nx < 2 || ny < 2 || nz < 2 || !F) return -1;
    const size_t N = (size_t)nx * ny * nz;
    const double* Fx = F; const double* Fy = F + N; const double* Fz = F + 2 * N;
    double* w = (double*)malloc(sizeof(double) * nz);
    if (!w) return -2;
    if (Qblend) {
        if (!QJ || !kaprho0 || !(tau0 > 0.0)) { free(w); return -1; }
        double tau = 0.0;
        for (int k = nz - 1; k >= 0; --k) {
            double s = 0.0;
            for (size_t n = 0; n < (size_t)nx * ny; ++n) s += kaprho0[(size_t)k * nx * ny + n];
            tau += s / ((double)nx * ny) * dz;
            w[k] = exp(-tau / tau0);
        }
    }
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                const size_t n = ((size_t)k * ny + j) * nx + i;
                const int ip = (i + 1) % nx, im = (i - 1 + nx) % nx;
                const int jp = (j + 1) % ny, jm = (j - 1 + ny) % ny;
                const int kp = (k + 1 < nz) ? k + 1 : k, km = (k > 0) ? k - 1 : k;
                const double dfx = (Fx[((size_t)k * ny + j) * nx + ip] - Fx[((size_t)k * ny + j) * nx + im]) / (2.0 * dx);
                const double dfy = (Fy[((size_t)k * ny + jp) * nx + i] - Fy[((size_t)k * ny + jm) * nx + i]) / (2.0 * dy);
                const double dfz = (Fz[((size_t)kp * ny + j) * nx + i] - Fz[((size_t)km * ny + j) * nx + i]) / (dz * (double)(kp - km));
                const double qd = -(dfx + dfy + dfz);
                if (Qdiv) Qdiv[n] = qd;
                if (Qblend) Qblend[n] = w[k] * QJ[n] + (1.0 - w[k]) * qd;
            }
    free(w);
    return 0;
}

/* ---------------------------------------------------------------------------
 * O-9  Grid staggering (paper's Interpolate, PAPER.md:79:
 *      "trilinear interpolation of the MHD variables from the MHD grid to the
 *      staggered RTS grid").  DESIGN.md reading R20: the MHD variables live at the
 *      centres of ncx*ncy*ncz cells, the RT nodes are the cell corners.  x and y are
 *      periodic, so there are nx = ncx, ny = ncy corner columns; there are
 *      nz = ncz + 1 corner levels, and below the bottom / above the top cell level
 *      the missing cells are the edge cells again (zero-gradient ghost level).
 *      Trilinear interpolation at a corner is the mean of its 8 cells:
 *        node(i,j,k) = 1/8 sum_{a,b,c in {0,1}} cell(wrap(i-a), wrap(j-b), clamp(k-c))
 *      O-1 holds for the result too: the node fields are fp32 arrays (the mean is
 *      formed in fp64 -- the sum of 8 floats is exact there -- and rounded once).
 * ------------------------------------------------------------------------- */
int oracle_cells_to_nodes(int ncx, int ncy, int ncz, const float* cell, float* node)
{
    if (ncx < 2 || ncy < 2 || ncz < 1 || !cell || !node) return -1;
    const int nz = ncz + 1;
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ncy; ++j)
            for (int i = 0; i < ncx; ++i) {
                double sum = 0.0;
                for (int c = 0; c < 2; ++c) {
                    int kk = k - c;
                    if (kk < 0) kk = 0;
                    if (kk > ncz - 1) kk = ncz - 1;
                    for (int b = 0; b < 2; ++b) {
                        const int jj = (j - b + ncy) % ncy;
                        for (int a = 0; a < 2; ++a) {
                            const int ii = (i - a + ncx) % ncx;
                            sum += (double)cell[((size_t)kk * ncy + jj) * ncx + ii];
                        }
                    }
                }
                node[((size_t)k * ncy + j) * ncx + i] = (float)(sum / 8.0);
            }
    return 0;
}

/* Heating back on the MHD grid: the mean of the 8 corner nodes of a cell,
 *   Qc(i,j,k) = 1/8 sum_{a,b,c in {0,1}} Qn(wrap(i+a), wrap(j+b), k+c),  k = 0..nz-2. */
int oracle_nodes_to_cells(int nx, int ny, int nz, const double* qn, double* qc)
{
    if (nx < 2 || ny < 2 || nz < 2 || !qn || !qc) return -1;
    for (int k = 0; k < nz - 1; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                double sum = 0.0;
                for (int c = 0; c < 2; ++c)
                    for (int b = 0; b < 2; ++b)
                        for (int a = 0; a < 2; ++a)
                            sum += qn[((size_t)(k + c) * ny + (j + b) % ny) * nx + (i + a) % nx];
                qc[((size_t)k * ny + j) * nx + i] = sum / 8.0;
            }
    return 0;
}

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
