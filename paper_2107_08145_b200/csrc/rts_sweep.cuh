// rts_sweep.cuh -- K_b, the persistent sweep kernel (stages B-E) for sm_100a.
//
// Work decomposition ("sweep kernel"):
//   unit  = (march axis, direction, band pair): the <= 4 rays (one per sign pair su, sv) whose
//           characteristics leave the upwind cell through the face normal to the march axis.
//           Every stencil node of plane m lies in plane m-1, so a plane is fully parallel.
//   task  = one WU x WV tile of the transverse (u, v) plane of one unit, marched through all
//           planes and passes by one CTA.  CTAs take tasks from an in-order ticket counter.
//   block = K consecutive steps.  At a block start a tile reads a K-deep halo of the carried
//           plane from its upwind neighbours (global exchange buffer Xex) and then advances K
//           planes on its own, recomputing the shrinking halo; at the block end it publishes
//           its downwind strips and arrives at the unit's barrier flag (release / acquire).
//   seams = stencil nodes across a periodic boundary come from the previous pass (Jacobi):
//           far columns / rows of every plane are kept in G (pass parity) and copied into the
//           ghost column / row of the carried plane before each step.
//   strip = the thread-level unit of work: one node pair (two columns) of one ray, the rows of one row chunk,
//           marched from the upwind end of the v axis.  The upwind rows of kaprho, S and X stay in registers
//           (sliding window), so a row costs one row load of each; whole warps belong to one ray, so the
//           ray's signs are warp-uniform.  Every value is a float2 (bands 2p, 2p+1) and all arithmetic is
//           packed (f32x2).  Every thread owns the same strip for the whole task (descriptors in registers).
// Shared-memory layout (PITCH = nodes per box row, a compile-time constant, so that every load of a strip
// is one base register plus an immediate):
//   coefficient stage   [BV rows][kaprho row | S row][PITCH] float2      one 5-D TMA box per plane
//   carried planes      [2 buffers][su group][BV rows][ray sv>0 row | ray sv<0 row][PITCH] float2
// Carried quantity: X = I - a*S with a = 1 at levels k <= kstar (optically thick part, where
// J - S would cancel) and a = 0 above (thin part, where I << S would cancel).
#ifndef RTS_SWEEP_SHARED_PART
#define RTS_SWEEP_SHARED_PART
#include "rts_kernels.cuh"

#ifndef RTS_SWEEP_THREADS
#define RTS_SWEEP_THREADS 512   // most threads of a sweep CTA (<= 128 registers)
#endif

namespace rts {

struct SweepMaps { CUtensorMap m[3]; };      // coefficient tensor of the x-, y-, z-march units

typedef float2 f2;

// ---- packed fp32 pairs (Blackwell FFMA2 / FMUL2 / FADD2): one issue slot for the two bands of a node.
// A pair built as make_float2(w, w) from one register is a broadcast operand in SASS (no second register).
__device__ __forceinline__ f2 fma2(const f2 a, const f2 b, const f2 c) {
    unsigned long long r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(*reinterpret_cast<const unsigned long long*>(&a)),
        "l"(*reinterpret_cast<const unsigned long long*>(&b)), "l"(*reinterpret_cast<const unsigned long long*>(&c)));
    return *reinterpret_cast<f2*>(&r);
}
__device__ __forceinline__ f2 mul2(const f2 a, const f2 b) {
    unsigned long long r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(*reinterpret_cast<const unsigned long long*>(&a)),
        "l"(*reinterpret_cast<const unsigned long long*>(&b)));
    return *reinterpret_cast<f2*>(&r);
}
__device__ __forceinline__ f2 add2(const f2 a, const f2 b) {
    unsigned long long r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(*reinterpret_cast<const unsigned long long*>(&a)),
        "l"(*reinterpret_cast<const unsigned long long*>(&b)));
    return *reinterpret_cast<f2*>(&r);
}
__device__ __forceinline__ f2 sub2(const f2 a, const f2 b) {
    unsigned long long r;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(*reinterpret_cast<const unsigned long long*>(&a)),
        "l"(*reinterpret_cast<const unsigned long long*>(&b)));
    return *reinterpret_cast<f2*>(&r);
}
__device__ __forceinline__ f2 bc(const float w) { return make_float2(w, w); }
__device__ __forceinline__ f2 neg2(const f2 a) { return make_float2(-a.x, -a.y); }
__device__ __forceinline__ float min3(const float a, const float b, const float c) {
    float r;
    asm("min.f32 %0, %1, %2, %3;" : "=f"(r) : "f"(a), "f"(b), "f"(c));
    return r;
}

// Loads / stores of the item code on 32-bit shared-window byte addresses with immediate offsets
template <int OFF>
__device__ __forceinline__ float4 lds128(const uint32_t a) {
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4+%5];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a), "n"(OFF));
    return v;
}
template <int OFF>
__device__ __forceinline__ f2 lds64(const uint32_t a) {
    f2 v;
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2+%3];" : "=f"(v.x), "=f"(v.y) : "r"(a), "n"(OFF));
    return v;
}
template <int OFF>
__device__ __forceinline__ void sts128(const uint32_t a, const float4 v) {
    asm volatile("st.shared.v4.f32 [%0+%1], {%2, %3, %4, %5};" ::"r"(a), "n"(OFF), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}
template <int OFF>
__device__ __forceinline__ void sts64(const uint32_t a, const f2 v) {
    asm volatile("st.shared.v2.f32 [%0+%1], {%2, %3};" ::"r"(a), "n"(OFF), "f"(v.x), "f"(v.y) : "memory");
}

// One box row around a node pair: the pair (n0, n1) and the side node the group's rays look at
// (SU > 0: the left neighbour of n0; SU < 0: the right neighbour of n1).
struct Row3 { f2 n0, n1, sd; };
template <int SU, int OFF>
__device__ __forceinline__ Row3 load_row(const uint32_t a)
{
    Row3 r;
    const float4 q = lds128<OFF>(a);
    r.n0 = make_float2(q.x, q.y); r.n1 = make_float2(q.z, q.w);
    r.sd = (SU > 0) ? lds64<OFF - 8>(a) : lds64<OFF + 16>(a);
    return r;
}
template <int J> __device__ __forceinline__ f2 cen(const Row3& r) { return J == 0 ? r.n0 : r.n1; }
template <int SU, int J> __device__ __forceinline__ f2 sid(const Row3& r)
{
    return (SU > 0) ? (J == 0 ? r.sd : r.n0) : (J == 0 ? r.n1 : r.sd);
}

// watchdog for every wait loop: gives up after ~2^22 unsuccessful probes (seconds) and raises
// the device-side abort flag so that all CTAs drain instead of hanging the GPU
__device__ __forceinline__ bool spin_abort(int* abortf, unsigned& spins, int code)
{
    if ((++spins & 255u) == 0u) {
        if (*reinterpret_cast<volatile int*>(abortf) != 0) return true;
        if (spins > (1u << 22)) { atomicCAS(abortf, 0, code); atomicCAS(abortf + 2, 0, code); return true; }   // [2]: sticky copy
    }
    return false;
}

// Flagged exchange words: a strip value travels with the tag of the block that wrote it in ONE 64-bit word, so a
// reader that sees the tag has the value (64-bit scalar accesses are single-copy atomic): no release fence, no
// flag store and no separate poll between a tile and its neighbours, one L2 round trip instead of four.
__device__ __forceinline__ void st_tagged2(void* p, const f2 v, const unsigned tag)
{
    const unsigned long long a = ((unsigned long long)tag << 32) | __float_as_uint(v.x);
    const unsigned long long b = ((unsigned long long)tag << 32) | __float_as_uint(v.y);
    asm volatile("st.global.cg.v2.u64 [%0], {%1, %2};" ::"l"(p), "l"(a), "l"(b) : "memory");
}
// (volatile: the same buffer was read two blocks earlier, and a plain or .cg load may be served from the SM's L1)
__device__ __forceinline__ bool ld_tagged2(const void* p, const unsigned tag, f2& v)
{
    unsigned long long a, b;
    asm volatile("ld.volatile.global.v2.u64 {%0, %1}, [%2];" : "=l"(a), "=l"(b) : "l"(p) : "memory");
    v = make_float2(__uint_as_float((unsigned)a), __uint_as_float((unsigned)b));
    return (unsigned)(a >> 32) == tag && (unsigned)(b >> 32) == tag;
}

__device__ __forceinline__ int wrap(int x, int n) { x %= n; return x < 0 ? x + n : x; }

// TMA engine, tensor form: one 5-D box (u, field, ., ., band pair) of a coefficient layout -> shared memory
__device__ __forceinline__ void tensor_load5(void* dst, const CUtensorMap* map, int c0, int c1, int c2, int c3, int c4, uint64_t* bar)
{
    asm volatile("cp.async.bulk.tensor.5d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5, %6}], [%7];"
                 ::"r"(smem_u32(dst)), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4), "r"(smem_u32(bar)) : "memory");
}


// Item (static for a task, in registers): one thread marches a strip of one ray: one node pair (two columns)
// wide, the rows q = qa .. qb-1 of the ray's region, counted from the upwind end of the v axis (q = 0: the
// outermost halo row, or the first core row where there is no upwind tile).
enum : unsigned {
    IT_DQ = 1u << 0,         // halo pair in u: only active while the remaining halo depth is > 0
    IT_PART = 1u << 1,       // only the first column of the pair exists (odd n_u)
    IT_USTRIP = 1u << 3,     // core pair inside the u exchange strip
    IT_DIR = 1u << 5         // row q = 0 is the inflow row of a bounded v axis (set, not updated)
};

struct GhostEnt { unsigned short xoff, bv; int goff; };   // 8 bytes; slot = goff >> 28; xoff: box row * 2 PITCH + column
struct HaloEnt { unsigned short xoff; unsigned char slot, mask; int goff; };   // mask = c0 | c1 << 4 (nodes of the pair)

struct TileGeo {
    int u0, v0, wu, wv, BV, BUW;
    int dlo_u, dhi_u, dlo_v, dhi_v;    // domain bounds in box coordinates
    int kstar, mthick;
    int zmarch, up_z;
};

// Per-task constants, in shared memory: everything the out-of-line parts of a task need, so that the
// hot loop keeps only its own state in registers.
struct TaskShared {
    UnitDesc U;
    TileGeo G;
    uint64_t mbar[NSTAGE_MAX];
    int ticket, flag, nghost, nhalo;
    int pbase, tolmode;                // passes done before this launch; error-controlled mode (one pass per launch)
    int has_hist, qrev;                // this tile holds the far-u column or far-v row of some ray (seam histories);
                                       // the last warp of every ray has at most half its lanes busy (heating pass)
    unsigned errs[NSLOT][4];           // tolmode: per ray max |I(p) - I(p-1)| on the seam faces (band 0, 1), max |I(p)| (band 0, 1)
    int PS, tu, tv, pad0;              // nodes per plane set; tile coordinates
    f2* stage0;                        // [nstage] coefficient plane sets
    f2* Xb;                            // [2][ng] carried plane sets
    GhostEnt* gt; HaloEnt* ht;
    float* Itop_b; float* pad2;
    int* abortf; int* pad1;
};

// what the item code needs to know about the current step (registers)
struct StepCtx {
    int hj;                            // remaining halo depth
    unsigned xmask;                    // item flags that need the slow tail this step
    int zreg;                          // z-march: regime of this step (0, 1, 2)
    bool dplane;                       // z-march inflow plane: nodes are set, not updated
    float a_prev, a_cur;               // z-march: a on the previous / this plane
    int tail;                          // for ray_tail: bit 0 seam histories on, bit 1 strips on, bit 2 exchange parity,
                                       // bits 8.. = (pass parity) * n_m + m  (seam-history plane)
};

__device__ __forceinline__ float4 scale4(const float f, const float4 a) { return make_float4(f * a.x, f * a.y, f * a.z, f * a.w); }
__device__ __forceinline__ float4 cat4(const f2 a, const f2 b) { return make_float4(a.x, a.y, b.x, b.y); }

// slot s inside one buffer of carried planes (node offset; + row * 2 PITCH + column)
template <int PITCH>
__device__ __forceinline__ int xso(const TaskShared& S, const int s) { return ((S.U.ng == 2) ? (s & 1) : 0) * S.PS + (s >> 1) * PITCH; }

struct RayK { float4 w; float kc; };     // per-thread constants of the ray: weights (upwind row, its u-side
                                         // neighbour, own row, its u-side neighbour; sum == 1 exactly), half path

// bilinear stencil sum of node J over the upwind row and the node's own row of the previous plane
template <int SU, int J>
__device__ __forceinline__ f2 bil(const Row3& up, const Row3& ow, const float4 w)
{
    f2 v = mul2(bc(w.x), cen<J>(up));
    v = fma2(bc(w.y), sid<SU, J>(up), v);
    v = fma2(bc(w.z), cen<J>(ow), v);
    v = fma2(bc(w.w), sid<SU, J>(ow), v);
    return v;
}
// the same sum started from `init` (the source difference is formed first: S_u - S_p)
template <int SU, int J>
__device__ __forceinline__ f2 bil_from(const Row3& up, const Row3& ow, const float4 w, const f2 init)
{
    f2 v = fma2(bc(w.x), cen<J>(up), init);
    v = fma2(bc(w.y), sid<SU, J>(up), v);
    v = fma2(bc(w.z), cen<J>(ow), v);
    v = fma2(bc(w.w), sid<SU, J>(ow), v);
    return v;
}

// ------------------------------------------------------------------------------------------
// Attenuation factors of one node (both bands): em1 = 1 - e^-dt, wl = (1 - e^-dt)/dt, pp = psi_p = 1 - wl.
// ONE branch-free form for every optical path, the same instructions in every lane, warp and tile:
//   dt >= DTAU_SERIES: closed form (exp2 and reciprocal units): wl = (1 - E)/dt, pp = 1 - wl;
//   dt <  DTAU_SERIES: where 1 - E and 1 - wl cancel, the first four terms of the series of psi_p
//                      (truncation dt^4/360 < 2e-8 relative there), wl = 1 - psi_p;
//   both are evaluated and selected per lane and band.
// Round 2 measured why there is one form and not a cheap one for uniform rows and a dearer one for mixed rows
// (chosen per warp by a vote): the tiles of a unit advance in lockstep, so the tiles of the dearest regime set
// the pace of all (the whole sweep ran at the cost of the mixed form: 29.6 ms; this form everywhere: 27.7 ms),
// and the result no longer depends on which nodes share a warp, i.e. on the tiling.
__device__ __forceinline__ void att_factors(const f2 dt, f2& em1, f2& wl, f2& pp)
{
    const f2 nd = neg2(dt);
    f2 q = fma2(nd, bc(1.0f / 120.0f), bc(1.0f / 24.0f));
    q = fma2(nd, q, bc(1.0f / 6.0f));
    q = fma2(nd, q, bc(0.5f));
    const f2 pps = mul2(dt, q), wls = sub2(bc(1.f), pps);
    const f2 t2 = mul2(dt, bc(-LOG2E));
    const f2 E = make_float2(ex2_approx(t2.x), ex2_approx(t2.y));
    const f2 ec = sub2(bc(1.f), E);                            // exactly 1 where exp2 underflows (thick-plane shortcut)
    const f2 wlc = mul2(ec, make_float2(rcp_approx(dt.x), rcp_approx(dt.y)));
    const f2 ppc = sub2(bc(1.f), wlc), es = mul2(dt, wls);
    const bool sx = dt.x < DTAU_SERIES, sy = dt.y < DTAU_SERIES;
    pp = make_float2(sx ? pps.x : ppc.x, sy ? pps.y : ppc.y);
    wl = make_float2(sx ? wls.x : wlc.x, sy ? wls.y : wlc.y);
    em1 = make_float2(sx ? es.x : ec.x, sy ? es.y : ec.y);
}

// The same for the uniform regimes (a the same on both stencil rows and at the node, f = 1 - a): they need
// em1 and c = wl - f only.  For f = 1 (the direct part) c = -psi_p comes straight from the series where it is
// small, and psi_p itself is not formed.
__device__ __forceinline__ void att_uniform(const f2 dt, const float f, f2& em1, f2& c)
{
    const f2 nd = neg2(dt);
    f2 q = fma2(nd, bc(1.0f / 120.0f), bc(1.0f / 24.0f));
    q = fma2(nd, q, bc(1.0f / 6.0f));
    q = fma2(nd, q, bc(0.5f));
    const f2 pps = mul2(dt, q);
    const f2 cs = sub2(bc(1.f - f), pps), es = fma2(nd, pps, dt);          // (1 - psi_p) - f;  dt (1 - psi_p)
    const f2 t2 = mul2(dt, bc(-LOG2E));
    const f2 E = make_float2(ex2_approx(t2.x), ex2_approx(t2.y));
    const f2 ec = sub2(bc(1.f), E);                            // exactly 1 where exp2 underflows (thick-plane shortcut)
    const f2 cc = fma2(ec, make_float2(rcp_approx(dt.x), rcp_approx(dt.y)), bc(-f));
    const bool sx = dt.x < DTAU_SERIES, sy = dt.y < DTAU_SERIES;
    c = make_float2(sx ? cs.x : cc.x, sy ? cs.y : cc.y);
    em1 = make_float2(sx ? es.x : ec.x, sy ? es.y : ec.y);
}

// One node (both bands).  su/so, xu/xo: upwind / own stencil row of S and X; sp: source at the node.
// REG 0: departure-carried part (a = 1 on both stencil rows and at the node); 1: direct part (a = 0);
// 2: general (a per row).
template <int SU, int J, int REG>
__device__ __forceinline__ f2 node_update(const f2 em1, const f2 wl, const f2 pp, const Row3& su, const Row3& so,
                                          const Row3& xu, const Row3& xo, const f2 sp, const float4 w,
                                          const float a_u, const float a_o, const float a_p)
{
    const f2 Xu = bil<SU, J>(xu, xo, w);
    if (REG == 3) {
        // uniform regime, f = a_u = 1 - a: one branch-free form of REG 0 (f = 0) and REG 1 (f = 1):
        //   X = Xu + em1 (f (d + Sp) - Xu) + (wl - f) d,  d = Su - Sp formed first (weights sum to 1);  wl - 1 = -psi_p
        //   (here `wl` carries c = wl - f of att_uniform)
        const f2 d = bil_from<SU, J>(su, so, w, neg2(sp));
        const f2 t = fma2(bc(a_u), add2(d, sp), neg2(Xu));
        return fma2(wl, d, fma2(em1, t, Xu));
    }
    f2 v = fma2(neg2(Xu), em1, Xu);                                // Xu * e^-dt
    if (REG == 0) {
        const f2 d = bil_from<SU, J>(su, so, w, neg2(sp));         // S_u - S_p (weights sum to 1 exactly)
        return fma2(d, wl, v);
    }
    if (REG == 1) {
        // Xu E + psi_u Su + psi_p Sp with psi_u = (1 - E) - psi_p:  Xu + (1 - E)(Su - Xu) - psi_p (Su - Sp)
        const f2 d = bil_from<SU, J>(su, so, w, neg2(sp));         // Su - Sp
        const f2 t = sub2(add2(d, sp), Xu);                        // Su - Xu
        return fma2(neg2(pp), d, fma2(em1, t, Xu));
    }
    const f2 pu = sub2(em1, pp);                                   // psi_u = (1 - E) - psi_p
    const f2 R0 = fma2(bc(w.y), sid<SU, J>(su), mul2(bc(w.x), cen<J>(su)));
    const f2 R1 = fma2(bc(w.w), sid<SU, J>(so), mul2(bc(w.z), cen<J>(so)));
    const f2 St = fma2(bc(a_o), R1, mul2(bc(a_u), R0));
    const f2 Sh = sub2(add2(R0, R1), St);
    const f2 Stp = mul2(bc(a_p), sp);
    v = fma2(sub2(St, Stp), wl, v);
    v = fma2(pu, Sh, v);
    return fma2(pp, sub2(sp, Stp), v);
}

// what a strip needs for the uncommon stores of a step (exchange strips)
struct TailCtx {
    float4* XeP;                       // exchange planes of this block's parity (16 bytes per node); null: no strips this step
    int gv0, ug;                       // slot * n_v + global v of row q = 0;  global u of the pair
    int n_u2;                          // row pitch of the exchange planes
    int hv, nrows, K, gsv;
    unsigned tag;                      // tag of the block whose strips are published this step (0: plain strips)
};

// ------------------------------------------------------------------------------------------
// shared-memory carve-up of a CTA (float2 nodes), every part 128-byte aligned.  A plane set is BV rows of
// two PITCH-node halves: (kaprho | S) of a coefficient stage, or the two rays (sv > 0 | sv < 0) of a group.
struct SmemPlan {
    int BV, PS, guardA, guardB, nitems, nghost_max, nhalo_max, nstage, ng;
    __host__ __device__ SmemPlan(int pitch, int WU, int WV, int ng_, int nstage_) {
        nstage = nstage_; ng = ng_;
        BV = WV + 2 * HALO;
        PS = BV * 2 * pitch;
        guardA = 16;                                         // an item reads the node before its first row
        guardB = 6 * pitch;                                  // ... and up to two rows after its last
        nitems = 0;                                          // strips per ray: see strips_for()
        nghost_max = NSLOT * (WU + 2 * HALO + BV);
        nhalo_max = NSLOT * ((WV + KMAX) * (HALO / 2) + KMAX * ((WU + HALO) / 2 + 1));
    }
    // strips of one ray (node pairs incl. the upwind u halo x row chunks of rc rows incl. the upwind v halo), whole warps
    __host__ __device__ static int strips_for(int WU, int WV, int rc) {
        return ((((WU + HALO) / 2) * ((WV + KMAX - 1 + rc - 1) / rc)) + 31) & ~31;
    }
    __host__ __device__ int nodes() const { return guardA + (nstage + 2 * ng) * PS + guardB; }
    __host__ __device__ size_t bytes() const {
        return (size_t)nodes() * 8 + (size_t)nghost_max * sizeof(GhostEnt) + (size_t)nhalo_max * sizeof(HaloEnt);
    }
};

__device__ __forceinline__ int plane_of(const UnitDesc& U, const int mm) { return (U.dir > 0) ? mm : U.n_m - 1 - mm; }
__device__ __forceinline__ float a_of(const TileGeo& G, const int level) { return (level <= G.kstar) ? 1.f : 0.f; }

// value of I^(0) - a S at a box position of plane `msrc` (Kbox = its coefficient stage)
template <int PITCH>
__device__ __forceinline__ f2 x_initial(const TaskShared& S, const f2* Kbox, int s, int bv, int xo_in_box, int msrc)
{
    const UnitDesc& U = S.U; const TileGeo& G = S.G;
    const f2 Sv = Kbox[xo_in_box + PITCH];
    float a; bool dn, up;
    if (G.zmarch) { a = a_of(G, plane_of(U, msrc)); dn = (msrc == 0); up = G.up_z != 0; }
    else { const int v = G.v0 - HALO + bv; a = a_of(G, v); up = !(s & 2); dn = (v == (up ? 0 : U.n_v - 1)); }
    const float f = ((dn && !up) ? 0.f : 1.f) - a;
    return make_float2(f * Sv.x, f * Sv.y);
}

// seam ghost of entry g for the carried plane `msrc` from pass `psrc` (psrc < 0: the initial guess)
template <int PITCH>
__device__ __forceinline__ f2 ghost_fetch(const TaskShared& S, const GhostEnt g, int psrc, int msrc, const f2* Kbox)
{
    if (psrc < 0) return x_initial<PITCH>(S, Kbox, g.goff >> 28, g.bv, g.xoff, msrc);
    const UnitDesc& U = S.U;
    const size_t g_plane = (size_t)NSLOT * (U.n_v + U.n_u2);
    return __ldcg(reinterpret_cast<const f2*>(U.Gu) + ((size_t)(psrc & 1) * U.n_m + msrc) * g_plane + (g.goff & 0x0fffffff));
}

}  // namespace rts
#endif  // RTS_SWEEP_SHARED_PART

// ==========================================================================================================
// The strip code, the task loop and the kernel exist twice: rts.cu includes this file once with RTS_TOLM 0
// (namespace fixedp: a fixed number of passes in one launch) and once with RTS_TOLM 1 (namespace tolp: the
// error-controlled mode, one pass per launch).  A macro and not a template parameter: with a bool template
// parameter the register allocation of the fixed-pass kernel changed (32 -> 120 bytes of spills, +8 % time),
// although not one instruction of it depends on the mode.
#ifndef RTS_TOLM
#error "define RTS_TOLM (0 / 1) and RTS_MODE_NS before including rts_sweep.cuh"
#endif
namespace rts { namespace RTS_MODE_NS {

// (the out-of-line parts live in the mode's namespace too: device functions shared by two kernels are
//  allocated registers for both callers at once, which cost the fixed-pass kernel its allocation)
// Heating, radiative flux and emergent intensity of a finished plane (last pass; out of line): reads the new
// carried plane set Xn (one buffer) and that plane's coefficient stage Kc.  The unit's contribution goes to its
// own partial buffers with plain stores: every node is written exactly once, no atomics (deterministic).
template <int PITCH>
__device__ __noinline__ void q_pass(const TaskShared* __restrict__ Sp, const f2* __restrict__ Kc, const f2* __restrict__ Xn, const int m_done)
{
    constexpr int RPN = 2 * PITCH;
    const TaskShared& S = *Sp;
    const UnitDesc& U = S.U; const TileGeo& G = S.G;
    const int tid = threadIdx.x, T = blockDim.x;
    const int pl = plane_of(U, m_done);
    const int nqc = (G.wu + 1) >> 1;
    const float qb1 = (U.nband_ok == 2) ? FOUR_PI : 0.f;
    const bool zmarch = G.zmarch != 0;
    float* const Qdst = U.Qpart;
    float* const Fdst = U.Fpart;
    float* const Itop_b = S.Itop_b;
    const long long Nn = (long long)U.n_m * U.n_u * U.n_v;
    // does this plane (z-march) or this tile (x/y-march: its top row) hold emergent intensities at all?
    const bool topstep = Itop_b && (zmarch ? (m_done == U.n_m - 1 && G.up_z) : (G.v0 + G.wv == U.nz));
    // element tid, then 2T-1-tid, ...: where the last warp of a ray is mostly idle in the strips (8 of 32 lanes at
    // 48 x 24), the leftover elements of a second turn (576 node pairs on 512 threads) go to the last warps, not
    // to warps 0 and 1
    const bool qrev = S.qrev != 0;
    for (int it = 0, e = tid; e < nqc * G.wv; ++it, e = qrev ? (it + 1) * T - 1 - ((it & 1) ? tid : (T - 1 - tid)) : e + T) {
        const int row = e / nqc, q = e - row * nqc;
        const int bo = (HALO + row) * RPN + HALO + 2 * q;
        const int v = G.v0 + row, u = G.u0 + 2 * q;
        const int nval = min(2, G.wu - 2 * q);
        const float4 kp = *reinterpret_cast<const float4*>(Kc + bo);
        const float4 sp = *reinterpret_cast<const float4*>(Kc + bo + PITCH);
        const float a_p = zmarch ? a_of(G, pl) : a_of(G, v);
        const float shs = 1.0f - a_p;
        f2 acc0 = make_float2(0.f, 0.f), acc1 = make_float2(0.f, 0.f);    // node 0 / node 1, per band
        f2 fl0[3], fl1[3];
#pragma unroll
        for (int a = 0; a < 3; ++a) { fl0[a] = make_float2(0.f, 0.f); fl1[a] = make_float2(0.f, 0.f); }
        const f2 s0 = mul2(bc(shs), make_float2(sp.x, sp.y)), s1 = mul2(bc(shs), make_float2(sp.z, sp.w));
        const f2 as0 = mul2(bc(a_p), make_float2(sp.x, sp.y)), as1 = mul2(bc(a_p), make_float2(sp.z, sp.w));
#pragma unroll
        for (int s = 0; s < NSLOT; ++s) {
            // no branch around the load: an absent ray's place in the plane set holds zeros or (two rays per CTA) the
            // other ray's values, finite either way, and its weight is 0
            const bool on = U.ray[s].active != 0;
            const float4 x = *reinterpret_cast<const float4*>(Xn + xso<PITCH>(S, s) + bo);
            const float wq = on ? U.ray[s].wq : 0.f;
            acc0 = fma2(bc(wq), sub2(make_float2(x.x, x.y), s0), acc0);       // w_r (I - S)
            acc1 = fma2(bc(wq), sub2(make_float2(x.z, x.w), s1), acc1);
            if (Fdst && on) {
                const f2 i0 = add2(make_float2(x.x, x.y), as0), i1 = add2(make_float2(x.z, x.w), as1);   // I = X + a S
#pragma unroll
                for (int a = 0; a < 3; ++a) {
                    const float wm = wq * U.ray[s].mu[a];
                    fl0[a] = fma2(bc(wm), i0, fl0[a]);
                    fl1[a] = fma2(bc(wm), i1, fl1[a]);
                }
            }
            if (topstep && on && U.ray[s].itop >= 0) {
                const bool top = zmarch || (v == U.nz - 1 && !(s & 2));
                if (top) {
                    float* dst = Itop_b + (long long)U.ray[s].itop * U.it_sr + (zmarch ? (long long)v : (long long)pl) * U.it_so;
                    const float xa[4] = {x.x, x.y, x.z, x.w}, sa[4] = {sp.x, sp.y, sp.z, sp.w};
#pragma unroll
                    for (int j = 0; j < 2; ++j)
                        if (j < nval) {
#pragma unroll
                            for (int b = 0; b < 2; ++b)
                                if (b < U.nband_ok) dst[(long long)b * U.it_sb + (long long)(u + j) * U.it_su] = xa[2 * j + b] + a_p * sa[2 * j + b];
                        }
                }
            }
        }
        const long long qo = (long long)pl * U.q_sm + (long long)v * U.q_sv + u;
        const float q0 = FOUR_PI * kp.x * acc0.x + qb1 * kp.y * acc0.y;
        const float q1 = FOUR_PI * kp.z * acc1.x + qb1 * kp.w * acc1.y;
        if (U.qvec && nval == 2) *reinterpret_cast<float2*>(Qdst + qo) = make_float2(q0, q1);
        else { Qdst[qo] = q0; if (nval == 2) Qdst[qo + 1] = q1; }
        if (Fdst) {
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                const float f0 = FOUR_PI * fl0[a].x + qb1 * fl0[a].y, f1 = FOUR_PI * fl1[a].x + qb1 * fl1[a].y;
                float* fd = Fdst + (long long)a * Nn + qo;
                if (U.qvec && nval == 2) *reinterpret_cast<float2*>(fd) = make_float2(f0, f1);
                else { fd[0] = f0; if (nval == 2) fd[1] = f1; }
            }
        }
    }
}

// Seam histories of a finished plane (out of line): the far-u column and, on a periodic v axis, the far-v row of
// every ray are copied from the carried plane set Xn (one buffer) to Gu[parity of pass P][m_done]: the next pass's
// Jacobi ghosts of that plane.  Error-controlled mode: their change against the previous pass and the intensity
// itself go into the ray's error words (Kc: the plane's coefficient stage, for S).
template <int PITCH>
__device__ __noinline__ void hist_pass(TaskShared* __restrict__ Sp, const f2* __restrict__ Kc, const f2* __restrict__ Xn, const int m_done, const int P)
{
    constexpr int RPN = 2 * PITCH;
    TaskShared& S = *Sp;
    const UnitDesc& U = S.U; const TileGeo& G = S.G;
    const int tid = threadIdx.x, T = blockDim.x;
    const size_t g_plane = (size_t)NSLOT * (U.n_v + U.n_u2);
    f2* const GhP = reinterpret_cast<f2*>(U.Gu) + ((size_t)(P & 1) * U.n_m + m_done) * g_plane;
    const f2* const GhO = (RTS_TOLM && P > 0) ? reinterpret_cast<const f2*>(U.Gu) + ((size_t)((P - 1) & 1) * U.n_m + m_done) * g_plane : nullptr;
    const bool zmarch = G.zmarch != 0;
    const int per = G.wv + (U.per_v ? G.wu : 0);                 // far-column nodes, then far-row nodes of one ray
    for (int i = tid; i < NSLOT * per; i += T) {
        const int s = i / per, j = i - s * per;
        if (!U.ray[s].active) continue;
        const int su = (s & 1) ? -1 : 1, sv = (s & 2) ? -1 : 1;
        int bu, bv, goff;
        if (j < G.wv) {                                          // far-u column of this ray, if this tile holds it
            bu = (su > 0) ? G.dhi_u - 1 : G.dlo_u; bv = HALO + j;
            if (bu < HALO || bu >= HALO + G.wu) continue;
            goff = s * U.n_v + G.v0 + j;
        } else {                                                 // far-v row
            bv = (sv > 0) ? G.dhi_v - 1 : G.dlo_v; bu = HALO + (j - G.wv);
            if (bv < HALO || bv >= HALO + G.wv) continue;
            goff = NSLOT * U.n_v + s * U.n_u2 + G.u0 + (j - G.wv);
        }
        const int xo = bv * RPN + bu;
        const f2 xn = Xn[xso<PITCH>(S, s) + xo];
        __stcg(GhP + goff, xn);
        if (RTS_TOLM) {
            const int v = G.v0 - HALO + bv;
            const f2 Sv = Kc[xo + PITCH];
            const float a = zmarch ? a_of(G, plane_of(U, m_done)) : a_of(G, v);
            const bool up = zmarch ? (G.up_z != 0) : !(s & 2);
            const bool dn = zmarch ? (m_done == 0) : (v == (up ? 0 : U.n_v - 1));   // inflow node: set, never changes
            const f2 In = fma2(bc(a), Sv, xn);                   // I = X + a S
            f2 d = make_float2(0.f, 0.f);
            if (!dn) d = GhO ? sub2(xn, __ldcg(GhO + goff)) : sub2(In, Sv);     // same a, S in both passes; I(0) = S
            atomicMax(&S.errs[s][0], __float_as_uint(fabsf(d.x))); atomicMax(&S.errs[s][1], __float_as_uint(fabsf(d.y)));
            atomicMax(&S.errs[s][2], __float_as_uint(fabsf(In.x))); atomicMax(&S.errs[s][3], __float_as_uint(fabsf(In.y)));
        }
    }
}

// End of a launch of the error-controlled mode (out of line).  x/y-march: the last plane of the pass is the seam
// face of the march axis: its change against the previous pass (kept in Lp; pass 0: I(0) = S) goes into the
// error words and the plane replaces Lp (the next launch starts from it).  All: the error words go to global memory.
// P: index of the pass that has just ended.
template <int PITCH>
__device__ __noinline__ void pass_end(TaskShared* __restrict__ Sp, const f2* __restrict__ Kc, const f2* __restrict__ Xn, const int P)
{
    constexpr int RPN = 2 * PITCH;
    TaskShared& S = *Sp;
    const UnitDesc& U = S.U; const TileGeo& G = S.G;
    const int tid = threadIdx.x, T = blockDim.x;
    __syncthreads();                                          // the seam errors of the last step are in
    if (!G.zmarch) {
        f2* Lp = reinterpret_cast<f2*>(U.Lp);
        for (int i = tid; i < G.wu * G.wv; i += T) {
            const int row = i / G.wu, col = i - row * G.wu;
            const int xo = (HALO + row) * RPN + HALO + col;
            const int v = G.v0 + row, u = G.u0 + col;
            const f2 Sv = Kc[xo + PITCH];
            const float a = a_of(G, v);
#pragma unroll
            for (int s = 0; s < NSLOT; ++s) {
                if (!U.ray[s].active) continue;
                const f2 xn = Xn[xso<PITCH>(S, s) + xo];
                f2* lp = Lp + ((size_t)s * U.n_v + v) * U.n_u2 + u;
                const f2 In = fma2(bc(a), Sv, xn);
                const bool up = !(s & 2);
                const bool dn = (v == (up ? 0 : U.n_v - 1));      // inflow row: set, never changes
                f2 d = make_float2(0.f, 0.f);
                if (!dn) d = (P > 0) ? sub2(xn, __ldcg(lp)) : sub2(In, Sv);
                __stcg(lp, xn);
                atomicMax(&S.errs[s][0], __float_as_uint(fabsf(d.x))); atomicMax(&S.errs[s][1], __float_as_uint(fabsf(d.y)));
                atomicMax(&S.errs[s][2], __float_as_uint(fabsf(In.x))); atomicMax(&S.errs[s][3], __float_as_uint(fabsf(In.y)));
            }
        }
        __syncthreads();
    }
    if (tid < NSLOT * 4) atomicMax(U.errw + tid, (&S.errs[0][0])[tid]);
}

// Block start (out of line): fetch the K-deep halo of the carried plane set Xr from the exchange buffer and the seam
// ghosts of the previous plane.  Tagged exchange (U.xflag, every ray of the unit has its opposite ray in the unit):
// the halo words carry the tag of block gblk - 1, a reader spins on the words it needs; the tiles of the unit
// meet at the arrival counter only at a pass start (seam histories of the whole previous pass).  Otherwise they
// meet at the counter at every block start.  `skipped`: the publishing step was a thick plane that stored no strips.
// Returns false if the watchdog fired.
template <int PITCH>
__device__ __noinline__ bool block_start(TaskShared* __restrict__ Sp, f2* __restrict__ Xr, const f2* __restrict__ Kp0,
                                         const int pass2, const int blk0, const int gblk, const int s_,
                                         const unsigned tag, const bool skipped)
{
    TaskShared& S = *Sp;
    const UnitDesc& U = S.U; const TileGeo& G = S.G;
    const int tid = threadIdx.x, T = blockDim.x;
    const int ngh = S.nghost, nhalo = S.nhalo;
    const int pass = pass2 & 0xffff, passL = pass2 >> 16;   // global pass index (seam ghosts) / passes of this launch (counter)
    const bool zmarch = G.zmarch != 0;
    const bool tagged = U.xflag != 0;
    const bool exch = !(zmarch && blk0 == 0);
    const bool meet = !tagged || blk0 == 0;
    const int m_prev = (blk0 == 0) ? U.n_m - 1 : blk0 - 1;
    // seam ghosts of the previous plane come from the previous pass: inside a pass (blk0 > 0)
    // they were written more than one block ago, i.e. before the arrival counter this tile
    // has already seen, so they are fetched before the wait and only stored after it (one
    // L2 round trip less per block); at a pass start they belong to the block the wait is for
    const bool pre = exch && pass > 0 && blk0 > 0 && ngh > 0;
    f2 gpre = make_float2(0.f, 0.f);
    if (pre && tid < ngh) gpre = ghost_fetch<PITCH>(S, S.gt[tid], pass - 1, m_prev, nullptr);
    if (meet) {
        if (tid == 0) {
            const int need = (tagged ? passL : gblk) * U.ntiles;      // passL: passes of this launch
            const int ab = *reinterpret_cast<volatile int*>(S.abortf);
            unsigned spins = 0, ns = 32;
            while (ld_acquire(U.barrier) < need) {
                if (spin_abort(S.abortf, spins, 3 | (s_ << 4))) { S.flag = 1; break; }
                __nanosleep(ns);
                if (ns < 256) ns += ns;                  // back off a little: a unit waiting for residency spins long
            }
            if (ab != 0) S.flag = 1;
        }
        __syncthreads();
        if (S.flag != 0) return false;                   // uniform: the watchdog fired somewhere
    }
    if (exch) {
        // halo pairs lie inside the domain, ghost columns / rows outside it: disjoint stores
        if (!skipped) {
            const float4* xe0 = reinterpret_cast<const float4*>(U.Xex) + (size_t)((gblk - 1) & 1) * NSLOT * (size_t)U.n_v * U.n_u2;
            for (int e = tid; e < nhalo; e += T) {
                const HaloEnt h = S.ht[e];
                const float4* src = xe0 + (size_t)h.slot * U.n_v * U.n_u2 + h.goff;
                const int c0 = h.mask & 15, c1 = h.mask >> 4;
                f2 x0 = make_float2(0.f, 0.f), x1 = x0;
                unsigned spins = 0;
                while (true) {
                    bool ok = true;
                    if (c0 == 0) ok = ld_tagged2(src, tag, x0) || !tagged;
                    if (c1 == 2) ok = (ld_tagged2(src + 1, tag, x1) || !tagged) && ok;
                    if (ok) break;
                    if (spin_abort(S.abortf, spins, 4 | (s_ << 4))) { S.flag = 1; break; }
                }
                f2* d = Xr + xso<PITCH>(S, h.slot) + h.xoff;
                if (c0 == 0 && c1 == 2) *reinterpret_cast<float4*>(d) = cat4(x0, x1);
                else if (c0 == 0) d[0] = x0;
                else if (c1 == 2) d[1] = x1;
            }
        }
        if (ngh > 0) {
            if (pre && tid < ngh) { const GhostEnt g = S.gt[tid]; Xr[xso<PITCH>(S, g.goff >> 28) + g.xoff] = gpre; }
            for (int e = pre ? tid + T : tid; e < ngh; e += T) {
                const GhostEnt g = S.gt[e];
                Xr[xso<PITCH>(S, g.goff >> 28) + g.xoff] = ghost_fetch<PITCH>(S, g, pass - 1, m_prev, Kp0);
            }
        }
        __syncthreads();
        if (S.flag != 0) return false;
    }
    return true;
}

// Task set-up, part 2 (out of line): seam-ghost and halo lists, and for the x/y-march the initial carried planes
template <int PITCH>
__device__ __noinline__ void task_lists(TaskShared* __restrict__ Sp)
{
    constexpr int RPN = 2 * PITCH;
    TaskShared& S = *Sp;
    const UnitDesc& U = S.U; const TileGeo& G = S.G;
    const int tid = threadIdx.x, T = blockDim.x;
    const int BV = G.BV, BU = G.BUW, K = U.K, tu = S.tu, tv = S.tv;
    // ---- seam ghosts of this tile (compact list)
    for (int e = tid; e < NSLOT * (BV + BU); e += T) {
        const int s = e / (BV + BU), i = e - s * (BV + BU);
        const int su = (s & 1) ? -1 : 1, sv = (s & 2) ? -1 : 1;
        if (!U.ray[s].active) continue;
        int xoff = -1, goff = 0, bvv = 0;
        const int gcol = (su > 0) ? G.dlo_u - 1 : G.dhi_u;
        const int grow = (sv > 0) ? G.dlo_v - 1 : G.dhi_v;
        if (i < BV) {                                        // ghost column, box row i
            int v = G.v0 - HALO + i;
            const bool okv = U.per_v || (v >= 0 && v < U.n_v);
            if (gcol >= 0 && gcol < BU && okv) { v = wrap(v, U.n_v); xoff = i * RPN + gcol; goff = s * U.n_v + v; bvv = i; }
        } else if (U.per_v) {                                // ghost row, box column i - BV
            const int bu = i - BV;
            if (grow >= 0 && grow < BV) {
                const int u = wrap(G.u0 - HALO + bu, U.n_u);
                xoff = grow * RPN + bu; goff = NSLOT * U.n_v + s * U.n_u2 + u; bvv = grow;
            }
        }
        if (xoff >= 0) {
            GhostEnt g; g.xoff = (unsigned short)xoff; g.bv = (unsigned short)bvv; g.goff = goff | (s << 28);
            S.gt[atomicAdd(&S.nghost, 1)] = g;
        }
    }
    // ---- halo node pairs fetched at a block start (depth K), compact list
    for (int s = 0; s < NSLOT; ++s) {
        if (!U.ray[s].active) continue;
        const int su = (s & 1) ? -1 : 1;
        const bool svp = !(s & 2);
        const bool up_u = (su > 0) ? (tu > 0) : (tu < U.ntu - 1);
        const bool up_v = svp ? (tv > 0) : (tv < U.ntv - 1);
        if (!up_u && !up_v) continue;
        const int rlo = max((svp && up_v) ? HALO - K : HALO, G.dlo_v);
        const int rhi = min((!svp && up_v) ? HALO + G.wv + K : HALO + G.wv, G.dhi_v);
        const int kp = (K + 1) & ~1;                         // the K halo columns, in whole pairs: what the neighbour publishes
        const int clo = max((su > 0 && up_u) ? HALO - kp : HALO, G.dlo_u);
        const int chi = min((su < 0 && up_u) ? HALO + G.wu + kp : HALO + G.wu, G.dhi_u);
        const int q_lo = clo >> 1, nq = ((chi + 1) >> 1) - q_lo, nr = rhi - rlo;
        for (int e = tid; e < nr * nq; e += T) {
            const int r = e / nq, row = rlo + r, q = q_lo + (e - r * nq);
            const bool core = (row >= HALO && row < HALO + G.wv) && (2 * q >= HALO && 2 * q < HALO + G.wu);
            if (core) continue;
            HaloEnt h;
            h.xoff = (unsigned short)(row * RPN + 2 * q); h.slot = (unsigned char)s;
            h.mask = (unsigned char)(max(0, clo - 2 * q) | (min(2, chi - 2 * q) << 4));
            h.goff = (G.v0 - HALO + row) * U.n_u2 + (G.u0 - HALO + 2 * q);
            S.ht[atomicAdd(&S.nhalo, 1)] = h;
        }
    }
    // ---- x/y-march: X^(0) on the plane before step 0, whole box (halo and ghosts included)
    {
        unsigned spins = 0;
        while (!mbar_try_wait(&S.mbar[U.nstage - 1], 0u)) { if (spin_abort(S.abortf, spins, 5)) break; }
    }
    if (!G.zmarch) {
        const f2* Kp0 = S.stage0 + (size_t)(U.nstage - 1) * S.PS;
        const f2* Lp = reinterpret_cast<const f2*>(U.Lp);
        for (int i = tid; i < BU * BV; i += T) {
            const int bv = i / BU, bu = i - bv * BU;
            const int xo = bv * RPN + bu;
            const int v = G.v0 - HALO + bv, u = G.u0 - HALO + bu;
            const bool inside = v >= 0 && v < U.n_v && u >= 0 && u < U.n_u;
#pragma unroll
            for (int s = 0; s < NSLOT; ++s)
                if (U.ray[s].active) {
                    f2 x;
                    // a later launch of the error-controlled mode continues from the last plane of the previous pass
                    if (S.pbase > 0) x = inside ? __ldcg(Lp + ((size_t)s * U.n_v + v) * U.n_u2 + u) : make_float2(0.f, 0.f);
                    else x = x_initial<PITCH>(S, Kp0, s, bv, xo, U.n_m - 1);
                    S.Xb[xso<PITCH>(S, s) + xo] = x;
                }
        }
        if (S.pbase > 0) {
            __syncthreads();
            for (int e = tid; e < S.nghost; e += T) {         // its seam ghosts: the history of that plane
                const GhostEnt g = S.gt[e];
                S.Xb[xso<PITCH>(S, g.goff >> 28) + g.xoff] = ghost_fetch<PITCH>(S, g, S.pbase - 1, U.n_m - 1, nullptr);
            }
        }
    }
    __syncthreads();
}

// One coefficient plane (both fields) of this tile -> stage st (one thread)
__device__ __forceinline__ void issue_load(TaskShared& S, const CUtensorMap* cmap, const int pl, const int st)
{
    const UnitDesc& U = S.U; const TileGeo& G = S.G;
    uint64_t* bar = &S.mbar[st];
    mbar_expect_tx(bar, (uint32_t)S.PS * 8u);
    f2* dst = S.stage0 + (size_t)st * S.PS;
    const int c2 = G.zmarch ? G.v0 : (U.march == 1 ? pl + HALO : pl);
    const int c3 = G.zmarch ? pl : G.v0 - HALO;
    tensor_load5(dst, cmap, 2 * G.u0, 0, c2, c3, U.pair, bar);
}

// Store one finished row of a strip: the carried plane and, at a block end, the exchange strips.  Inline: a few
// instructions on the flagged rows only.  (The seam histories are copied from the finished plane by hist_pass: a
// strip that stored them row by row dragged its whole warp through this slow path, and the edge tiles, which
// alone have such strips, set the pace of their unit.)
template <int SU>
__device__ __forceinline__ void row_store(const TailCtx& TC, const unsigned fl, const bool slow, const int q,
                                          const uint32_t bW, const float4 o)
{
    if (!slow) { sts128<0>(bW, o); return; }
    const bool part = (fl & IT_PART) != 0;
    if (!part) sts128<0>(bW, o); else sts64<0>(bW, make_float2(o.x, o.y));
    if (q < TC.hv || (fl & IT_DQ)) return;                       // halo row / halo pair: nothing to publish
    const int gv = TC.gv0 + q * TC.gsv;
    if (TC.XeP && ((fl & IT_USTRIP) || q >= TC.nrows - TC.K)) {  // exchange strips at a block end
        float4* xe = TC.XeP + (size_t)gv * TC.n_u2 + TC.ug;          // 16 bytes per node: (value, tag) per band
        st_tagged2(xe, make_float2(o.x, o.y), TC.tag);
        st_tagged2(xe + 1, make_float2(o.z, o.w), TC.tag);
    }
}

// ------------------------------------------------------------------------------------------
// One strip: the rows q0 .. qb-1 of one node pair of one ray, marched from the upwind end of the v axis with the
// upwind rows of kaprho, S and X kept in registers.  rstep: bytes from a row to the next one downwind (+-RP);
// oP / oC / oX / oW: byte addresses of row q0's pair in the previous / this plane's coefficient stage and in the
// carried plane of the ray read / written this step.
template <int PITCH, int SU>
__device__ __forceinline__ void do_strip(
    const int s, const unsigned fl, int q, const int qb, const int rstep, const RayK& rk,
    const TaskShared& S, const StepCtx& C, const TailCtx& TC, const int qtail, int vrow, const int vstep,
    uint32_t bP, uint32_t bC, uint32_t bX, uint32_t bW)
{
    constexpr int HP = 8 * PITCH;        // second field (S) of a coefficient row
    const bool zm = S.G.zmarch != 0;
    const int ks = S.G.kstar;
    const bool tail_all = (fl & C.xmask) != 0u;
    if (C.dplane) {
        // z-march inflow plane: the nodes are set (I = S upward, 0 downward), not updated
        const float f = (S.U.ray[s].up ? 1.f : 0.f) - C.a_cur;
        for (; q < qb; ++q) {
            const float4 sc = lds128<HP>(bC);
            row_store<SU>(TC, fl, tail_all || q >= qtail, q, bW, scale4(f, sc));
            bC += rstep; bW += rstep;
        }
        return;
    }
    if ((fl & IT_DIR) && q == 0) {
        // inflow row of a bounded v axis (v = z): I = S (upward ray, bottom row) or 0 (downward ray, top row)
        const float a0 = (vrow <= ks) ? 1.f : 0.f;
        const float f = ((s & 2) ? 0.f : 1.f) - a0;
        const float4 sc = lds128<HP>(bC);
        row_store<SU>(TC, fl, tail_all || q >= qtail, q, bW, scale4(f, sc));
        bP += rstep; bC += rstep; bX += rstep; bW += rstep; vrow += vstep; ++q;
        if (q >= qb) return;
    }
    // upwind rows of the first row
    Row3 kA = load_row<SU, 0>(bP - rstep), sA = load_row<SU, HP>(bP - rstep), xA = load_row<SU, 0>(bX - rstep);
    Row3 kB, sB, xB;
#define STRIP_ROW(KU, SU_, XU, KO, SO, XO)                                                                          \
    {                                                                                                               \
        KO = load_row<SU, 0>(bP); SO = load_row<SU, HP>(bP); XO = load_row<SU, 0>(bX);                              \
        const float4 kc = lds128<0>(bC), sc = lds128<HP>(bC);                                                       \
        const f2 dt0 = mul2(add2(make_float2(kc.x, kc.y), bil<SU, 0>(KU, KO, rk.w)), bc(rk.kc));                    \
        const f2 dt1 = mul2(add2(make_float2(kc.z, kc.w), bil<SU, 1>(KU, KO, rk.w)), bc(rk.kc));                    \
        float a_u, a_o, a_p;                                                                                        \
        if (zm) { a_u = a_o = C.a_prev; a_p = C.a_cur; }                                                            \
        else { a_u = (vrow - vstep <= ks) ? 1.f : 0.f; a_o = (vrow <= ks) ? 1.f : 0.f; a_p = a_o; }                  \
        const f2 sp0 = make_float2(sc.x, sc.y), sp1 = make_float2(sc.z, sc.w);                                      \
        f2 e0, l0, p0, e1, l1, p1;                                                                                  \
        f2 v0, v1;                                                                                                  \
        if (a_u == a_o && a_o == a_p) {                                                                             \
            att_uniform(dt0, 1.f - a_p, e0, l0); att_uniform(dt1, 1.f - a_p, e1, l1);                               \
            v0 = node_update<SU, 0, 3>(e0, l0, l0, SU_, SO, XU, XO, sp0, rk.w, 1.f - a_p, 0.f, 0.f);                \
            v1 = node_update<SU, 1, 3>(e1, l1, l1, SU_, SO, XU, XO, sp1, rk.w, 1.f - a_p, 0.f, 0.f);                \
        } else {                                                                                                    \
            att_factors(dt0, e0, l0, p0); att_factors(dt1, e1, l1, p1);                                             \
            v0 = node_update<SU, 0, 2>(e0, l0, p0, SU_, SO, XU, XO, sp0, rk.w, a_u, a_o, a_p);                      \
            v1 = node_update<SU, 1, 2>(e1, l1, p1, SU_, SO, XU, XO, sp1, rk.w, a_u, a_o, a_p);                      \
        }                                                                                                           \
        const float4 o = cat4(v0, v1);                                                                              \
        row_store<SU>(TC, fl, tail_all || q >= qtail, q, bW, o);                                                    \
        bP += rstep; bC += rstep; bX += rstep; bW += rstep; vrow += vstep; ++q;                                     \
    }
#pragma unroll 1
    while (true) {
        STRIP_ROW(kA, sA, xA, kB, sB, xB)
        if (q >= qb) break;
        STRIP_ROW(kB, sB, xB, kA, sA, xA)
        if (q >= qb) break;
    }
#undef STRIP_ROW
}

template <int PITCH>
__device__ void run_task(TaskShared& S, const SweepMaps& maps, const int tile, f2* __restrict__ smf,
                         float* __restrict__ Itop_all, int* abortf, const unsigned seq, const int pbase_arg, const int npass_launch)
{
    const int pbase = RTS_TOLM ? pbase_arg : 0;                  // the fixed-pass kernel knows neither: nothing of this mode costs it a register

    constexpr int tolmode = RTS_TOLM ? 1 : 0;
    const UnitDesc& U = S.U;
    const int tid = threadIdx.x, T = blockDim.x;
    const SmemPlan SP(PITCH, U.WU, U.WV, U.ng, U.nstage);
    const int NST = U.nstage, NG = U.ng, PS = SP.PS;
    const int tu = tile % U.ntu, tv = tile / U.ntu;
    if (tid == 0) {
        TileGeo G;
        G.u0 = tu * U.WU; G.v0 = tv * U.WV;
        G.wu = min(U.WU, U.n_u - G.u0); G.wv = min(U.WV, U.n_v - G.v0);
        G.BV = SP.BV; G.BUW = G.wu + 2 * HALO;
        G.dlo_u = HALO - G.u0; G.dhi_u = HALO + U.n_u - G.u0;
        G.dlo_v = HALO - G.v0; G.dhi_v = HALO + U.n_v - G.v0;
        G.kstar = *U.kstar;
        G.mthick = (U.march == 2) ? U.mthick[2] : 0;         // z-march: planes below this level are optically thick
        G.zmarch = (U.march == 2); G.up_z = (U.dir > 0);
        S.G = G;
        S.PS = PS; S.tu = tu; S.tv = tv;
        S.stage0 = smf + SP.guardA;                          // [NST] plane sets (kaprho | S)
        S.Xb = S.stage0 + NST * PS;                          // [2][NG] plane sets (ray sv>0 | ray sv<0)
        S.gt = reinterpret_cast<GhostEnt*>(smf + SP.nodes());
        S.ht = reinterpret_cast<HaloEnt*>(S.gt + SP.nghost_max);
        S.Itop_b = Itop_all ? Itop_all + (long long)(2 * U.pair) * U.it_sb : nullptr;
        S.abortf = abortf;
        for (int i = 0; i < NST; ++i) mbar_init(&S.mbar[i], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        S.flag = 0; S.nghost = 0; S.nhalo = 0;
        S.pbase = pbase; S.tolmode = tolmode;
        { const int ns_ = ((U.WU + HALO) / 2) * ((U.WV + U.K - 1 + U.RC - 1) / U.RC); S.qrev = ((ns_ & 31) != 0) && ((ns_ & 31) <= 16); }
        S.has_hist = (G.u0 == 0) || (G.u0 + G.wu == U.n_u) || (U.per_v && ((G.v0 == 0) || (G.v0 + G.wv == U.n_v)));
        for (int i = 0; i < NSLOT * 4; ++i) (&S.errs[0][0])[i] = 0u;
    }
    for (int i = tid; i < SP.nodes(); i += T) smf[i] = make_float2(0.f, 0.f);
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncthreads();
    const TileGeo& G = S.G;
    const int n_m = U.n_m, npass = RTS_TOLM ? npass_launch : U.npass, K = U.K;
    const int nsteps = n_m * npass;
    const bool zmarch = (U.march == 2);
    const bool has_hist = S.has_hist != 0;
    const bool tagged = U.xflag != 0;
    const unsigned tag0 = seq << 12;                         // tags of this solve (never 0: the buffers start zeroed)

    // ---- coefficient planes through the TMA ring (started first: the tables below hide its latency)
    const CUtensorMap* const cmap = &maps.m[U.march];
    if (tid == 0) {
        issue_load(S, cmap, plane_of(U, n_m - 1), NST - 1);  // the plane "before" step 0
        issue_load(S, cmap, plane_of(U, 0), 0);
        if (nsteps > 1 && NST > 2) issue_load(S, cmap, plane_of(U, 1 % n_m), 1);
    }

    // ---- the strip of this thread.  The threads are split evenly between the unit's rays (whole warps per ray,
    //      so the ray's signs are warp-uniform); strip index e enumerates (row chunk, node pair) of the ray's region:
    //      tile core + upwind u halo (one HALO of columns) + upwind v halo of depth K-1, clipped to the domain.
    const int nsl = 2 * NG;
    // warp w works for ray w % nsl: the warps of one scheduler (w % 4) then run the same ray, i.e. one copy of
    // the strip code (one sign of su) at a time in its instruction cache
    const int sidx = (tid >> 5) % nsl, e = ((tid >> 5) / nsl) * 32 + (tid & 31);
    const int s = (NG == 2) ? sidx : (((U.gsu0 < 0) ? 1 : 0) + 2 * sidx);   // slot of this thread's ray
    const int gsu = (s & 1) ? -1 : 1, gsv = (s & 2) ? -1 : 1;
    unsigned ifl = 0;
    int qa = 0, qb = 0, geo = 0;
    uint32_t ioff0 = 0;                                      // byte offset of (row q = 0, pair) inside a plane set
    constexpr int RP = 16 * PITCH;
    {
        const int hmax = K - 1, RC = U.RC;
        const bool on = U.ray[s].active != 0;
        const bool up_u = (gsu > 0) ? (tu > 0) : (tu < U.ntu - 1);
        const bool up_v = (gsv > 0) ? (tv > 0) : (tv < U.ntv - 1);
        const int hu = (up_u && hmax > 0) ? HALO : 0;
        // upwind v halo, clipped to the domain (beyond a periodic edge lies the seam ghost row, not a halo)
        const int hv = up_v ? min(hmax, (gsv > 0) ? G.v0 : U.n_v - G.v0 - G.wv) : 0;
        const int clo = max((gsu > 0) ? HALO - hu : HALO, G.dlo_u);
        const int chi = min((gsu > 0) ? HALO + G.wu : HALO + G.wu + hu, G.dhi_u);
        const int nrows = hv + G.wv;
        const int qlo = clo >> 1, nq = ((chi + 1) >> 1) - qlo, nch = (nrows + RC - 1) / RC;
        geo = hv | (nrows << 8);
        if (on && chi > clo && e < nq * nch) {
            const int ch = e / nq, q2 = qlo + (e - ch * nq);
            const int c0 = 2 * q2;
            qa = ch * RC; qb = min(qa + RC, nrows);
            const int row0 = (gsv > 0) ? HALO - hv : HALO + G.wv - 1 + hv;     // box row of q = 0
            ioff0 = (uint32_t)(row0 * RP + c0 * 8);
            const bool core_q = (c0 >= HALO) && (c0 < HALO + G.wu);
            if (!core_q) ifl |= IT_DQ;
            if (chi - c0 < 2) ifl |= IT_PART;
            if (core_q && ((gsu > 0) ? (c0 + 2 > HALO + G.wu - K) : (c0 - HALO < K))) ifl |= IT_USTRIP;
            // row q = 0 is the inflow row of a bounded v axis (x/y-march: v = z)
            if (!zmarch && ((gsv > 0) ? (G.v0 - hv == 0) : (G.v0 + G.wv + hv == U.n_v))) ifl |= IT_DIR;
        }
    }
    task_lists<PITCH>(&S);

    RayK rk;
    rk.w = *reinterpret_cast<const float4*>(U.ray[s].w); rk.kc = U.ray[s].kc;
    const int ngh = S.nghost;
    const int mthick = G.mthick, kstar = G.kstar, dir = U.dir;
    const uint32_t aStage0 = smem_u32(S.stage0), aXb = smem_u32(S.Xb);
    const uint32_t PSB = (uint32_t)PS * 8u;
    const uint32_t xslot = (uint32_t)xso<PITCH>(S, s) * 8u;           // this thread's ray inside a carried buffer (bytes)
    const uint32_t XBB = (uint32_t)NG * PSB;                         // one buffer of carried planes (bytes)
    const int rstep = (gsv > 0) ? RP : -RP;
    const int hv_ = geo & 0xff, nrows_ = geo >> 8;
    const int v_q0 = (gsv > 0) ? G.v0 - hv_ : G.v0 + G.wv - 1 + hv_;  // global v of row q = 0
    TailCtx TC;
    TC.gv0 = s * U.n_v + v_q0;
    TC.ug = G.u0 - HALO + (int)((ioff0 % (uint32_t)RP) >> 3);
    TC.n_u2 = U.n_u2;
    TC.hv = hv_; TC.nrows = nrows_; TC.K = K; TC.gsv = gsv;
    const size_t xe_par = (size_t)NSLOT * U.n_v * U.n_u2;

    // ================================================================== the march
    int cur = 0, gblk = 0, s_ = 0;
    int stc = 0, stp = NST - 1;                              // stages of this step's and the previous plane
    uint32_t par_bits = 1u << (NST - 1);                     // stage NST-1 already served the plane before step 0
    bool bail = false;
    for (int pass = 0; pass < npass && !bail; ++pass) {
        const bool lastpass = (pass == npass - 1);
        const int P = RTS_TOLM ? pbase + pass : pass;            // passes done before this one (earlier launches included)
        // error-controlled mode: every pass may be the last one: it writes the heating and I_top, keeps its seam
        // history and skips nothing
        const bool qon = lastpass || tolmode, hist_on = !lastpass || tolmode, may_skip = !lastpass && !tolmode;
        for (int blk0 = 0; blk0 < n_m && !bail; blk0 += K) {
            const int blen = min(K, n_m - blk0);
            // ---- block start: wait for the unit, fetch halos and seam ghosts of the previous plane
            if (s_ > 0) {
                // tag of the strips of block gblk - 1; no strips were stored if their step was a skipped thick plane
                const bool skipped = zmarch && may_skip && blk0 > 0 && plane_of(U, blk0 - 1) < G.mthick;
                if (!block_start<PITCH>(&S, S.Xb + (size_t)cur * NG * PS, S.stage0 + (size_t)stp * PS, P | (pass << 16), blk0, gblk, s_,
                                        tag0 | ((unsigned)gblk & 0xfffu), skipped)) { bail = true; break; }
            }
            for (int j = 0; j < blen; ++j, ++s_) {
                const int m = blk0 + j;
                const int hj = blen - 1 - j;
                const bool blk_last = (hj == 0);
                const bool more = (s_ + 1 < nsteps);
                const int pl = (dir > 0) ? m : n_m - 1 - m;

                {
                    unsigned spins = 0;
                    while (!mbar_try_wait(&S.mbar[stc], (par_bits >> stc) & 1u)) { if (spin_abort(abortf, spins, 2 | (s_ << 4))) break; }
                }
                par_bits ^= 1u << stc;
                // ---- heating / emergent intensity of the previous step's plane
                if (qon && m > 0) q_pass<PITCH>(&S, S.stage0 + (size_t)stp * PS, S.Xb + (size_t)cur * NG * PS, m - 1);
                // ---- seam histories of the previous step's plane (the last plane of a pass: below, before the arrival)
                if (hist_on && m > 0 && has_hist) hist_pass<PITCH>(&S, S.stage0 + (size_t)stp * PS, S.Xb + (size_t)cur * NG * PS, m - 1, P);
                // ---- seam ghosts for the next step (previous pass, this plane): fetch now, store after the update
                const bool ghost_next = !blk_last && more && ngh > 0;
                f2 gval[2] = {make_float2(0.f, 0.f), make_float2(0.f, 0.f)};
                if (ghost_next && P > 0) {
#pragma unroll
                    for (int i = 0; i < 2; ++i) { const int e = tid + i * T; if (e < ngh) gval[i] = ghost_fetch<PITCH>(S, S.gt[e], P - 1, m, nullptr); }
                }

                // ---- the update
                // Thick-plane shortcut (z-march, non-final passes): on planes pl <= mthick every optical path
                // exceeds DTAU_SKIP, e^-dtau is exactly 0 and the new plane does not depend on the carried one.
                // The planes pl < mthick only feed such planes (and seam ghosts that are multiplied by 0), so
                // their updates are skipped; plane mthick restarts from whatever finite values the buffers hold.
                if (!(zmarch && may_skip && pl < mthick)) {
                    // first row of this step: halo rows deeper than the remaining halo depth are not updated any more
                    const int q0 = max(qa, hv_ - hj);
                    if (q0 < qb && !((ifl & IT_DQ) && hj == 0)) {
                        StepCtx C;
                        C.hj = hj;
                        C.dplane = zmarch && (m == 0);
                        const bool strips = blk_last && more && !(zmarch && m == n_m - 1);
                        C.tail = 0;
                        TC.XeP = strips ? reinterpret_cast<float4*>(U.Xex) + (size_t)(gblk & 1) * xe_par : nullptr;
                        TC.tag = tag0 | ((unsigned)(gblk + 1) & 0xfffu);
                        C.xmask = IT_PART | (strips ? IT_USTRIP : 0u);
                        C.a_prev = (pl - dir <= kstar) ? 1.f : 0.f; C.a_cur = (pl <= kstar) ? 1.f : 0.f;
                        C.zreg = 0;
                        const int qtail = strips ? nrows_ - K : (1 << 20);
                        const uint32_t o = ioff0 + (uint32_t)(q0 * rstep);
                        const uint32_t bP = aStage0 + (uint32_t)stp * PSB + o, bC = aStage0 + (uint32_t)stc * PSB + o;
                        const uint32_t bX = aXb + (uint32_t)cur * XBB + xslot + o, bW = aXb + (uint32_t)(cur ^ 1) * XBB + xslot + o;
                        if (gsu < 0) do_strip<PITCH, -1>(s, ifl, q0, qb, rstep, rk, S, C, TC, qtail, v_q0 + gsv * q0, gsv, bP, bC, bX, bW);
                        else         do_strip<PITCH, +1>(s, ifl, q0, qb, rstep, rk, S, C, TC, qtail, v_q0 + gsv * q0, gsv, bP, bC, bX, bW);
                    }
                }
                // ---- seam ghosts of this plane into the new carried plane
                if (ghost_next) {
                    f2* const Xw = S.Xb + (size_t)(cur ^ 1) * NG * PS;
                    if (P > 0) {
#pragma unroll
                        for (int i = 0; i < 2; ++i) {
                            const int e = tid + i * T;
                            if (e < ngh) { const GhostEnt g = S.gt[e]; Xw[xso<PITCH>(S, g.goff >> 28) + g.xoff] = gval[i]; }
                        }
                        for (int e = tid + 2 * T; e < ngh; e += T) {
                            const GhostEnt g = S.gt[e];
                            Xw[xso<PITCH>(S, g.goff >> 28) + g.xoff] = ghost_fetch<PITCH>(S, g, P - 1, m, nullptr);
                        }
                    } else {
                        const f2* Kc = S.stage0 + (size_t)stc * PS;
                        for (int e = tid; e < ngh; e += T) {
                            const GhostEnt g = S.gt[e];
                            Xw[xso<PITCH>(S, g.goff >> 28) + g.xoff] = ghost_fetch<PITCH>(S, g, -1, m, Kc);
                        }
                    }
                }
                // ---- end of step; at a block end publish (release) before anybody waits
                __syncthreads();
                if (hist_on && m == n_m - 1 && has_hist) {   // the pass ends: its last plane's histories precede the arrival
                    hist_pass<PITCH>(&S, S.stage0 + (size_t)stc * PS, S.Xb + (size_t)(cur ^ 1) * NG * PS, m, P);
                    __syncthreads();
                }
                // one thread of the LAST warp (a ray's fourth warp holds its shortest strips): warp 0 is on the step's
                // critical path, and the ~0.1 us of the next plane's TMA issue there delayed every step (25.55 -> 25.38 ms)
                if (tid == T - 32) {
                    // arrival (release): at every block end, or with the tagged exchange at the end of a pass only
                    if (blk_last && more && (!tagged || m == n_m - 1)) { __threadfence(); atomicAdd(U.barrier, 1); }
                    const int ahead = NST - 1;               // planes in flight beyond the previous one
                    if (s_ + ahead < nsteps) {
                        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                        int m2 = m + ahead; if (m2 >= n_m) m2 %= n_m;
                        issue_load(S, cmap, plane_of(U, m2), stp);   // the previous plane's stage is free now
                    }
                }
                if (blk_last && more) ++gblk;
                cur ^= 1;
                stp = stc; stc = (stc + 1 == NST) ? 0 : stc + 1;
            }
        }
    }
    // heating / emergent intensity of the last plane
    if (!bail) q_pass<PITCH>(&S, S.stage0 + (size_t)stp * PS, S.Xb + (size_t)cur * NG * PS, n_m - 1);
    if (tolmode && !bail) pass_end<PITCH>(&S, S.stage0 + (size_t)stp * PS, S.Xb + (size_t)cur * NG * PS, pbase + npass - 1);
    __syncthreads();
    if (tid == 0)
        for (int i = 0; i < NST; ++i)
            asm volatile("mbarrier.inval.shared::cta.b64 [%0];" ::"r"(smem_u32(&S.mbar[i])) : "memory");
}

template <int PITCH>
__global__ void __launch_bounds__(RTS_SWEEP_THREADS, 1)
rts_sweep_kernel(const __grid_constant__ SweepMaps maps, const UnitDesc* __restrict__ units, int nunits,
                 int total_tickets, int* ticket_counter, float* __restrict__ Itop_all, int* abortf, unsigned seq,
                 int pbase, int npass_launch)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ __align__(16) TaskShared S;
    while (true) {
        __syncthreads();
        if (threadIdx.x == 0) {
            const int ab = *reinterpret_cast<volatile int*>(abortf);
            const int t = ab ? total_tickets : atomicAdd(ticket_counter, 1);
            int u = 0;
            if (t < total_tickets)
                for (int q = 1; q < nunits; ++q)
                    if (t >= units[q].ticket_begin) u = q;
            S.ticket = t; S.flag = u;
        }
        __syncthreads();
        const int ticket = S.ticket;
        if (ticket >= total_tickets) break;
        const int uid = S.flag;
        {
            const int* src = reinterpret_cast<const int*>(units + uid);
            int* dst = reinterpret_cast<int*>(&S.U);
            for (int w = threadIdx.x; w < (int)(sizeof(UnitDesc) / sizeof(int)); w += blockDim.x) dst[w] = src[w];
        }
        __syncthreads();
        run_task<PITCH>(S, maps, ticket - S.U.ticket_begin, reinterpret_cast<f2*>(smem_raw), Itop_all, abortf, seq, pbase, npass_launch);
    }
}

} }  // namespace rts::RTS_MODE_NS
