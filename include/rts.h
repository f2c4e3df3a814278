/*
 * rts.h -- C-ABI of the B200-native radiation transport solver (RTS) hot path.
 *
 * The operation is MURaM's RTS as described in arxiv 2107.08145:
 *   PAPER.md:78-82  (sec. 2)    RTS = Interpolate / Integrate / Exchange / Flux
 *   PAPER.md:189    (sec. 5.1)  short characteristics: integrate the transfer equation
 *                               along a ray using intensity and opacity interpolated from
 *                               the neighbouring grid cells, 3 rays per octant (24 rays)
 *   PAPER.md:195    (sec. 5.1)  multi-band opacities; boundary intensities iterated;
 *                               radiative heating/cooling at each point
 *   PAPER.md:197-217 (Fig. 8)   loop nest  rays x { interpol; iterate integrate; flux }
 * The numerical readings the paper leaves open are fixed in DESIGN.md ("Readings").
 *
 * One solve computes, for `nbands` opacity bands and `nrays` directions,
 *   stage A (interpol):  kaprho_b = 10^(bilinear log10 kappa_b(log10 T, log10 P)) * rho,
 *                        S_b = f_b(log10 T) * sigma T^4 / pi
 *   stage B (integrate): per ray and band the short-characteristics formal solution
 *                        I_p = I_u e^-dtau + psi_u S_u + psi_p S_p (linear source function),
 *                        upwind values bilinear on the entry face of the upwind cell,
 *                        dtau = (kaprho_u + kaprho_p)/2 * ds
 *   stage C:             `npasses` sweeps; a stencil node whose x or y index wraps around the
 *                        periodic box takes its intensity from the previous pass
 *                        (pass 0: I = S; inflow planes: bottom I = S, top I = 0)
 *   stage D (flux):      Q_rad = 4 pi sum_b kaprho_b (J_b - S_b),  J_b = sum_r w_r I_{b,r}
 *   stage E:             I_top[b][u] = I_{b,r}(.,.,nz-1) for the u-th ray with mu_z > 0
 *
 * Conventions
 *   - extern "C"; every function returns int: 0 = RTS_OK, negative = error.  No exceptions,
 *     no aborts, nothing printed.  rts_last_error() gives the text of the last failure.
 *   - Fields are fp32, contiguous [nz][ny][nx] (x fastest), z up, k = 0 is the bottom.  cgs.
 *   - "host"/"device" is stated per pointer.  The caller owns every buffer it passes in,
 *     including the device workspace; the library owns only small device copies of the
 *     tables and its job descriptors (freed by rts_destroy).  Inputs are never modified;
 *     outputs are fully overwritten (Q_rad is not accumulated into).
 *   - There is no CPU fallback: without a CUDA device rts_create fails with RTS_ECUDA.
 *   - Non-finite or non-positive T, P (log10 of <= 0) are the caller's responsibility.
 */
#ifndef RTS_H_
#define RTS_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define RTS_OK       0
#define RTS_EINVAL  -1   /* null pointer, bad size, bad ray, workspace too small or misaligned */
#define RTS_ESTATE  -2   /* call out of order (solve before tables / workspace) */
#define RTS_ECUDA   -3   /* CUDA runtime / launch error, or no device */
#define RTS_ENOMEM  -4   /* host allocation failed */
#define RTS_ETIMEOUT -5  /* device-side watchdog of the persistent sweep kernel fired */

typedef struct rts_ctx rts_ctx;

/* [PAPER.md:78-82, 189: the RTS on a 3-D Cartesian block; 3 rays per octant]
 * Create a solver for an nx*ny*nz node grid with spacings dx,dy,dz (cm) and nbands bands.
 * nx, ny >= 2 (periodic), nz >= 2, nbands >= 1.  Uses the current CUDA device.
 * Defaults: 24-ray set of BASELINE.json configs[0] (order: r = 3*octant + axis of the large
 * cosine, octant = bx + 2 by + 4 bz, b = 1 for a negative cosine; weights 1/24), 3 passes. */
int rts_create(rts_ctx** out, int nx, int ny, int nz,
               double dx_cm, double dy_cm, double dz_cm, int nbands);
int rts_destroy(rts_ctx* ctx);

/* [PAPER.md:195 "multi-band opacity scheme"; PAPER.md:79 interpol(); readings R8, R9]
 * Opacity and band-fraction tables; HOST pointers, copied to the device inside the call.
 *   logkappa[b][iT][iP] (iP fastest) = log10 kappa_b on a uniform nT x nP grid in
 *   (log10 T, log10 P) spanning [logT_min, logT_max] x [logP_min, logP_max]; lookups are
 *   bilinear with clamping at the edges.  bandfrac[b][iT] = f_b on the same log10 T grid
 *   (gray: all 1).  nT, nP >= 2. */
int rts_set_tables(rts_ctx* ctx, int nT, int nP,
                   double logT_min, double logT_max, double logP_min, double logP_max,
                   const float* logkappa_host, const float* bandfrac_host);

/* [PAPER.md:72 "iterated 3-4 times", Fig. 8: the while loop around integrate(); R11, R12]
 * Number of sweep passes (periodic re-sweeps with Jacobi seams), >= 1.  Default 3. */
int rts_set_passes(rts_ctx* ctx, int npasses);

/* [PAPER.md:189 "a set of 3 rays per octant are used to integrate over the unit sphere"; R2, R3]
 * Replace the ray set.  mu_xyz: HOST [nrays][3] directions of photon travel (need not be
 * normalised; mu_z must be non-zero); weights: HOST [nrays] (J = sum_r w_r I_r).
 * 1 <= nrays <= 256.  Invalidates the workspace size (call rts_workspace_bytes again). */
int rts_set_rays(rts_ctx* ctx, int nrays, const double* mu_xyz_host, const double* weights_host);
/* Read back the ray set (HOST out pointers may be NULL). *nrays receives the count. */
int rts_get_rays(const rts_ctx* ctx, int* nrays, double* mu_xyz_host, double* weights_host);
/* Number of rays with mu_z > 0 (second extent of I_top). */
int rts_num_up_rays(const rts_ctx* ctx);

/* [PAPER.md:221-239: integrate() is the hot spot; its wavefront is re-organised as a plane march, DESIGN.md 7.2]
 * Tuning hooks (optional).  march = 0,1,2 selects the sweeps that march along x, y, z.  A sweep
 * tile is tile_u nodes of the unit-stride transverse axis (rounded up to a multiple of 4,
 * <= 248) times tile_v nodes of the other transverse axis (<= 120); 0 = the planner's choice.
 * Tiles exchange halos every `steps` planes (1..4; 0 = default 4) and recompute a halo of that
 * depth in between.  ctas_per_sm = 0 lets the planner choose: two CTAs of <= 384 threads per SM, or
 * one CTA of <= 768 threads on a larger tile (1 or 2 force it).  All three invalidate
 * the workspace size (call rts_workspace_bytes / rts_set_workspace again). */
int rts_set_tiling(rts_ctx* ctx, int march, int tile_u, int tile_v);
int rts_set_exchange_interval(rts_ctx* ctx, int steps);
int rts_set_ctas_per_sm(rts_ctx* ctx, int ctas_per_sm);
/* Depth of the shared-memory ring the coefficient planes stream through: 3 (the load of the next plane
 * overlaps the current step), 2 (smaller footprint: larger tiles or two CTAs per SM), 0 = planner's choice. */
int rts_set_ring_depth(rts_ctx* ctx, int stages);

/* [PAPER.md:249-251: transposed copies of the coefficient arrays -- here two layouts in this workspace, DESIGN.md 6]
 * Bytes of device workspace the current configuration needs (0 on error). */
size_t rts_workspace_bytes(rts_ctx* ctx);
/* Hand over a DEVICE workspace of at least rts_workspace_bytes(), 256-byte aligned.  It must
 * stay valid until the ctx is destroyed or another workspace is set. */
int rts_set_workspace(rts_ctx* ctx, void* workspace_dev, size_t bytes);

/* [PAPER.md:197-217 Fig. 8: interpol(); iterate { integrate(); exchange } ; flux() -- stages A-E above]
 * The hot path.  DEVICE pointers: rho, T, P in [nz][ny][nx]; Qrad out [nz][ny][nx];
 * Itop out [nbands][n_up][ny][nx] or NULL (not wanted).  Qrad must be 16-byte aligned.  stream: a cudaStream_t passed as
 * void* (NULL = default stream).  Asynchronous on that stream; errors of the asynchronous
 * part surface at the next rts_sync_check / synchronising call. */
int rts_solve(rts_ctx* ctx, const float* rho_dev, const float* T_dev, const float* P_dev,
              float* Qrad_dev, float* Itop_dev, void* stream);

/* Radiative flux and flux-divergence heating (paper's Flux: "From the specific intensity calculate the average
 * intensity and radiative fluxes"; reading R21).  rts_enable_flux(1) must precede
 * rts_workspace_bytes / rts_set_workspace (three more partial fields per sweep unit).  rts_solve_flux is rts_solve plus
 *   Frad   DEVICE out [3][nz][ny][nx]: F_a = 4 pi sum_b sum_r w_r Omega_{r,a} I_{b,r}, Omega = mu/|mu| (band-integrated)
 *   Qdiv   DEVICE out [nz][ny][nx] or NULL: -div F, central differences on the node grid, periodic in x and y,
 *          one-sided on the bottom and top node planes
 *   Qblend DEVICE out [nz][ny][nx] or NULL: w Qrad + (1 - w) Qdiv, w(k) = exp(-taubar(k)/tau0), taubar(k) = horizontally
 *          averaged optical depth of band 0 from the top down to level k; tau0 set by rts_set_flux_blend (default 0.1).
 * Asynchronous on `stream`.  All sums are formed in a fixed order: results are bitwise reproducible. */
int rts_enable_flux(rts_ctx* ctx, int on);
int rts_set_flux_blend(rts_ctx* ctx, double tau0);
int rts_solve_flux(rts_ctx* ctx, const float* rho_dev, const float* T_dev, const float* P_dev,
                   float* Qrad_dev, float* Itop_dev, float* Frad_dev, float* Qdiv_dev, float* Qblend_dev, void* stream);

/* [same operation as rts_solve; the end-to-end entry bench.py's `e2e` times]
 * Same solve with HOST buffers (pinned or pageable): copies rho,T,P to the device, solves,
 * copies Qrad (and Itop if non-NULL) back, synchronises.  The staging buffers live in the
 * workspace (rts_workspace_bytes accounts for them).  The inputs travel in 8 slabs of levels on an internal
 * second stream while stage A follows slab by slab on `stream`; I_top goes back while the finalize kernel runs. */
int rts_solve_host(rts_ctx* ctx, const float* rho_host, const float* T_host, const float* P_host,
                   float* Qrad_host, float* Itop_host, void* stream);

/* Grid staggering (paper's Interpolate: "trilinear interpolation of the MHD variables from the MHD
 * grid to the staggered RTS grid"; reading R20).  The MHD variables live at
 * the centres of nx*ny*(nz-1) cells, the RT nodes of this ctx are the cell corners: x, y periodic,
 * the corner levels below / above the box repeat the edge cell level.
 *   rts_cells_to_nodes  node = correctly rounded mean of the 8 cells around a corner;
 *                       DEVICE cell [nz-1][ny][nx] -> DEVICE node [nz][ny][nx]
 *   rts_nodes_to_cells  cell = mean of its 8 corner nodes; DEVICE [nz][ny][nx] -> DEVICE [nz-1][ny][nx]
 *   rts_solve_cells     staggers rho, T, P (DEVICE, cell-centred [nz-1][ny][nx]) into the staging
 *                       part of the workspace, runs rts_solve on the node grid and averages Q_rad
 *                       back: Qrad_cells DEVICE out [nz-1][ny][nx]; Itop as in rts_solve.
 * Asynchronous on `stream`; inputs are not modified; needs tables and workspace like rts_solve. */
int rts_cells_to_nodes(rts_ctx* ctx, const float* cell_dev, float* node_dev, void* stream);
int rts_nodes_to_cells(rts_ctx* ctx, const float* node_dev, float* cell_dev, void* stream);
int rts_solve_cells(rts_ctx* ctx, const float* rho_cells_dev, const float* T_cells_dev, const float* P_cells_dev,
                    float* Qrad_cells_dev, float* Itop_dev, void* stream);

/* [PAPER.md:79, 204 interpol(); DESIGN.md 1 row A]
 * Stage A alone, for per-stage parity: DEVICE outputs kaprho, S each [nbands][nz][ny][nx]. */
int rts_coefficients(rts_ctx* ctx, const float* rho_dev, const float* T_dev, const float* P_dev,
                     float* kaprho_dev, float* S_dev, void* stream);

/* [no paper passage: error reporting of the persistent kernel of DESIGN.md 7.2]
 * Synchronise `stream` and report the device-side status of the solves since the last check
 * (RTS_OK, RTS_ETIMEOUT if the sweep watchdog fired in any of them -- the status is sticky until read --, RTS_ECUDA). */
int rts_sync_check(rts_ctx* ctx, void* stream);

/* [SURVEY 7, lever 4.ii; only the seam intensities change between the iterations]
 * Thick-plane shortcut (default on).  Where every optical path of a z-march ray on a level pair
 * exceeds 88.5 the fp32 exp underflows to exactly 0 and the update does not depend on the carried
 * intensity; the sweeps along z skip those planes in the non-final passes.  Results are bit-identical
 * for I_top and for Q_rad in the final pass (the heating is summed in a fixed order, no atomics).
 * rts_thick_levels: after a solve, HOST out [nbands] = number of level pairs from the bottom that were
 * found thick (synchronises `stream`); skipped updates = levels * nx * ny * (z-march rays) * (passes-1). */
int rts_set_thick_skip(rts_ctx* ctx, int on);
int rts_thick_levels(rts_ctx* ctx, int* levels_host, void* stream);

/* Error-controlled iteration and warm start (Fig. 8 "while(g_maxerr >
 * THRESHOLD) { ... integrate(); ... exchange(); err = error(); MPI_Allreduce(&err, &g_maxerr); }"
 * "iterates the intensities at the boundaries ... until the errors are within a prescribed tolerance";
 * DESIGN.md reading R22).  rts_set_tolerance(tol, max_passes) with max_passes >= 1 replaces the fixed pass
 * count: a solve sweeps one pass per kernel launch and stops after the first pass p for which, for every
 * (band, ray),   max over the two periodic seam faces |I(p) - I(p-1)|  <=  tol * max over them |I(p)|
 * (I(0) = S), or after max_passes passes; tol < 0 never stops early.  Q_rad and I_top are those of the last
 * pass run.  The solve is then SYNCHRONOUS on `stream` (the host reads the error words after every pass).
 * max_passes = 0 switches back to rts_set_passes.  Call before sizing the workspace (the mode keeps the last
 * plane of the x- and y-march sweeps in the workspace).
 * rts_set_warm_start(1): the next solves do not start from I(0) = S on the seam faces but from the faces the
 * previous solve on this context ended with (previous time step), as the paper's block-local solve does.
 * rts_passes_used: HOST outputs (either may be NULL): passes of the last solve, largest relative change of its
 * last pass.  RTS_ESTATE when the mode is off. */
int rts_set_tolerance(rts_ctx* ctx, double tol, int max_passes);
int rts_set_warm_start(rts_ctx* ctx, int on);
int rts_passes_used(rts_ctx* ctx, int* passes_host, float* relerr_last_host);

/* Band x octant sharding of ONE box over several GPUs ("for N-bands ... run N
 * times", PAPER.md:291 strong scaling of one 288^3 box).  The sweep units -- (march axis, direction, band
 * pair), i.e. the rays of one octant face group for two bands -- are dealt round robin to `nranks` contexts,
 * one per GPU / process.  After rts_set_shard(rank, nranks) a solve computes stage A for the whole box, sweeps
 * only this rank's units and returns PARTIAL results: Qrad = the heating of this rank's units, I_top = this
 * rank's (band, ray) slices, zeros elsewhere.  The caller completes both with one sum all-reduce over the ranks
 * (NCCL; paper_2107_08145_b200/multi.py).  Call before sizing the workspace (it changes the plan).
 * rts_shard_info: HOST outputs, units of this rank / of the whole problem.  RTS_EINVAL unless 0 <= rank < nranks. */
int rts_set_shard(rts_ctx* ctx, int rank, int nranks);
int rts_shard_info(rts_ctx* ctx, int* units_mine, int* units_all);

/* Scattering source function with the source update along the ray ("it is
 * preferable to use a Gauss-Seidel convergence scheme.  As the intensity is integrated along the ray, this scheme
 * will require updating the source function for each point along the ray, and then using the 'new' source function
 * to integrate the intensity at the next point along the ray"; reading R23).  For each of `nbands`
 * independent bands:
 *     S = (1 - eps) J + eps B,   J = sum_r w_r I_r,
 * kaprho, B (the thermal source), eps (photon destruction probability, 0 < eps <= 1): DEVICE float
 * [nbands][nz][ny][nx], e.g. the output of rts_coefficients (nbands need not be the context's band count).
 * Start S = B; every iteration visits the context's rays in index order, the planes of a ray along its exit-face
 * axis in upwind order, and at every node forms the short-characteristic intensity from the CURRENT S, then
 * (gauss_seidel != 0) J += w_r (I_new - I_old), S = (1 - eps) J + eps B at once, or (gauss_seidel == 0, the
 * Jacobi / Lambda iteration) S from all rays after the last one.  The periodic seams take one Jacobi pass per
 * iteration.  The bands share every plane step (and its grid barrier).  niter iterations, 0 <= niter <= 65536.
 * Outputs: S, J DEVICE double [nbands][nz][ny][nx] (this kernel computes in fp64); change_host (HOST
 * [niter][nbands], may be NULL): max|S - S_previous| / max|S| of every iteration and band.  workspace: DEVICE,
 * 256-byte aligned, at least rts_scatter_workspace_bytes(ctx, nbands, niter) bytes (one double per ray, node and
 * band, plus copies of the three inputs: 4.9 GB per band at 288^3 with 24 rays), borrowed for the call.  Synchronous on `stream` (the host reads
 * the change words).  RTS_ETIMEOUT if the grid barrier's watchdog fired; RTS_EINVAL for bad arguments. */
size_t rts_scatter_workspace_bytes(rts_ctx* ctx, int nbands, int niter);
int rts_scatter_solve(rts_ctx* ctx, int nbands, const float* kaprho_dev, const float* B_dev, const float* eps_dev,
                      int niter, int gauss_seidel, void* workspace_dev, size_t workspace_bytes, double* S_dev,
                      double* J_dev, double* change_host, void* stream);

/* The scattering solve for callers that cannot allocate device memory (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): the same operation, kernel and results as rts_scatter_solve (PAPER.md:261,
 * reading R23), with the scratch in a static device array of RTS_SCATTER_STATIC_BYTES bytes inside the library, which
 * every GPU that loads the library holds until the process exits.  The call makes no cudaMalloc / cudaFree and no
 * host heap allocation.  Arguments as rts_scatter_solve (inputs DEVICE float [nbands][nz][ny][nx], outputs DEVICE
 * double of the same shape, change_host HOST [niter][nbands] or NULL), without the workspace pair.
 * Limits: rts_scatter_workspace_bytes(ctx, nbands, niter) <= RTS_SCATTER_STATIC_BYTES (about 75 000 nodes x bands with
 * 24 rays), max(niter, 1) * nbands <= 2048, at most 256 rays; beyond them RTS_EINVAL with a message that names the
 * sizes.  The context's device must be current (RTS_ESTATE otherwise).  Every call on a device shares the one array,
 * which keeps the last call's contents (the entry clears what must start at zero): calls that overlap on the GPU
 * -- two streams, two contexts, two threads -- race; serialise them.  Synchronous on `stream`. */
#define RTS_SCATTER_STATIC_BYTES (16u << 20)
int rts_scatter_solve_static(rts_ctx* ctx, int nbands, const float* kaprho_dev, const float* B_dev, const float* eps_dev,
                             int niter, int gauss_seidel, double* S_dev, double* J_dev, double* change_host, void* stream);

/* [measurement only]
 * Per-stage device timing of the last rts_solve (CUDA events recorded on the solve stream
 * inside rts_solve).  rts_last_timing waits for the solve and fills ms4 (HOST) with
 * [0] stage A + switch heights, [1] all sweep launches, [2] finalize, [3] whole solve. */
int rts_enable_timing(rts_ctx* ctx, int on);
int rts_last_timing(rts_ctx* ctx, float* ms4_host);

/* [measurement only]
 * Plan facts for reporting: what[0] = kernels launched per solve, [1] = sweep tasks (tiles of
 * all units), [2] = CTAs per SM of the sweep kernel, [3] = sweep units (march axis x direction
 * x ray group x band), [4] = threads per CTA, [5] = dynamic shared memory per CTA (bytes),
 * [6] = sweep grid (persistent CTAs), [7] = exchange interval, [8..10] = tile_v of march x,y,z,
 * [11..13] = tile_u of march x,y,z, [14] = rays that march along z (leave their cell through a z face),
 * [15] = sweep units of the whole problem (= [3] unless sharded).  n = ints in `what` (<= 16). */
int rts_plan_info(rts_ctx* ctx, int* what, int n);

const char* rts_last_error(const rts_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* RTS_H_ */
