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
//   group = the rays of a unit with the same su (at most two: sv = +1, -1).  The warps of a CTA are
//           split between the groups, so su is warp-uniform.
//   item  = a 2 x 2 node block of one group: the thread-level unit of work.  Every thread owns the
//           same (at most two) items for the whole task; their descriptors live in registers.
//           The (kaprho, S) neighbourhood of an item is loaded once and serves both rays and both
//           bands: every value is a float2 (bands 2p, 2p+1) and all arithmetic is packed (f32x2).
// Per step a CTA streams one (kaprho, S) plane box through a TMA ring (one cp.async.bulk.tensor
// per field, completing on an mbarrier) and updates its items from registers and shared memory.
// Carried quantity: X = I - a*S with a = 1 at levels k <= kstar (optically thick part, where
// J - S would cancel) and a = 0 above (thin part, where I << S would cancel).
#pragma once
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

// Loads / stores of the item code on 32-bit shared-window byte addresses
__device__ __forceinline__ float4 lds128(const uint32_t a) {
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a));
    return v;
}
template <int OFF>
__device__ __forceinline__ f2 lds64(const uint32_t a) {
    f2 v;
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2+%3];" : "=f"(v.x), "=f"(v.y) : "r"(a), "n"(OFF));
    return v;
}
__device__ __forceinline__ void sts128(const uint32_t a, const float4 v) {
    asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(a), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}
__device__ __forceinline__ void sts64(const uint32_t a, const f2 v) {
    asm volatile("st.shared.v2.f32 [%0], {%1, %2};" ::"r"(a), "f"(v.x), "f"(v.y) : "memory");
}

// One box row around a node pair: the pair (n0, n1) and the side node the group's rays look at
// (SU > 0: the left neighbour of n0; SU < 0: the right neighbour of n1).
struct Row3 { f2 n0, n1, sd; };
template <int SU>
__device__ __forceinline__ Row3 load_row(const uint32_t a)
{
    Row3 r;
    const float4 q = lds128(a);
    r.n0 = make_float2(q.x, q.y); r.n1 = make_float2(q.z, q.w);
    r.sd = (SU > 0) ? lds64<-8>(a) : lds64<16>(a);
    return r;
}
template <int J> __device__ __forceinline__ f2 cen(const Row3& r) { return J == 0 ? r.n0 : r.n1; }
template <int SU, int J> __device__ __forceinline__ f2 sid(const Row3& r)
{
    return (SU > 0) ? (J == 0 ? r.sd : r.n0) : (J == 0 ? r.n1 : r.sd);
}
// bilinear stencil sum of node J: w = (lower v row, its side, higher v row, its side)
template <int SU, int J>
__device__ __forceinline__ f2 bil(const Row3& lo, const Row3& hi, const float4 w)
{
    f2 v = mul2(bc(w.x), cen<J>(lo));
    v = fma2(bc(w.y), sid<SU, J>(lo), v);
    v = fma2(bc(w.z), cen<J>(hi), v);
    v = fma2(bc(w.w), sid<SU, J>(hi), v);
    return v;
}
// the same sum started from `init` (the source difference is formed first: S_u - S_p)
template <int SU, int J>
__device__ __forceinline__ f2 bil_from(const Row3& lo, const Row3& hi, const float4 w, const f2 init)
{
    f2 v = fma2(bc(w.x), cen<J>(lo), init);
    v = fma2(bc(w.y), sid<SU, J>(lo), v);
    v = fma2(bc(w.z), cen<J>(hi), v);
    v = fma2(bc(w.w), sid<SU, J>(hi), v);
    return v;
}

__device__ __forceinline__ void red_add2(float* p, const float a, const float b)
{
    asm volatile("red.relaxed.gpu.global.add.v2.f32 [%0], {%1, %2};" ::"l"(p), "f"(a), "f"(b) : "memory");
}

// watchdog for every wait loop: gives up after ~2^22 unsuccessful probes (seconds) and raises
// the device-side abort flag so that all CTAs drain instead of hanging the GPU
__device__ __forceinline__ bool spin_abort(int* abortf, unsigned& spins, int code)
{
    if ((++spins & 255u) == 0u) {
        if (*reinterpret_cast<volatile int*>(abortf) != 0) return true;
        if (spins > (1u << 22)) { atomicCAS(abortf, 0, code); return true; }
    }
    return false;
}

__device__ __forceinline__ int wrap(int x, int n) { x %= n; return x < 0 ? x + n : x; }

// TMA engine, tensor form: one 4-D box (u, ., ., field) of a coefficient layout -> shared memory
__device__ __forceinline__ void tensor_load4(void* dst, const CUtensorMap* map, int c0, int c1, int c2, int c3, uint64_t* bar)
{
    asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
                 ::"r"(smem_u32(dst)), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(smem_u32(bar)) : "memory");
}


// Item descriptor (three registers, static for a task): pos = node offset in the box | first node
// row << 16 | node pair << 24; one flag word per ray of the group (sv > 0, sv < 0).  The item is
// the 2 x 2 node block (rows rowN, rowN+1; columns 2*pair, 2*pair+1).
enum : unsigned {
    IT_D0_SH = 2,            // bits 2-4   halo depth of node row 0 for this ray (0: core side; 7: never active)
    IT_D1_SH = 5,            // bits 5-7   halo depth of node row 1
    IT_DQ = 1u << 8,         // halo pair in u: only active while the remaining halo depth is > 0
    IT_REG_SH = 11,          // bits 11-12 regime of the stencil rows (x/y-march; static)
    IT_DIR0 = 1u << 13,      // node row is the inflow row of a bounded v axis
    IT_DIR1 = 1u << 14,
    IT_CORE0 = 1u << 15,     // node row and pair belong to the tile core
    IT_CORE1 = 1u << 16,
    IT_C1_SH = 19,           // bits 19-20 valid columns of the pair (1..2)
    IT_SPECIAL = 1u << 22,   // core item holding the far-v row of a periodic v axis: writes the seam history
    IT_STRIP0 = 1u << 23,    // core node row lies in an exchange strip
    IT_STRIP1 = 1u << 24,
    IT_FARC = 1u << 26       // core item holding the far-u column of its group: writes the seam history
};
constexpr unsigned IT_NEVER = (7u << IT_D0_SH) | (7u << IT_D1_SH);
constexpr int MAXIT = 2;     // items per thread

struct GhostEnt { unsigned short xoff, bv; int goff; };   // 8 bytes; slot = goff >> 28; xoff: node offset in the box
struct HaloEnt { unsigned short xoff; unsigned char slot, mask; int goff; };   // mask = c0 | c1 << 4 (nodes of the pair)

struct TaskShared {
    UnitDesc U;
    uint64_t mbar[NSTAGE_MAX];
    int ticket, flag, nghost, nhalo, pad0, pad1;
};

struct StepCtx {
    int hj, par_ex;                    // remaining halo depth, exchange parity
    int zreg;                          // z-march: regime of this step (0, 1, 2)
    bool dplane;                       // z-march inflow plane: nodes are set, not updated
    bool hist, strips;                 // write seam histories / publish strips this step
    float a_prev, a_cur;               // z-march: a on the previous / this plane
    f2* Ghist;                         // seam history of this plane and pass (far columns, then far rows)
};

struct TileGeo {
    int u0, v0, wu, wv, BU, BV, BOXN;
    int dlo_u, dhi_u, dlo_v, dhi_v;    // domain bounds in box coordinates
    int kstar;
    bool zmarch;
};

// plane of slot s among the carried planes of a CTA (units with one ray group keep two planes)
__device__ __forceinline__ int xplane(const UnitDesc& U, const int s) { return U.ng == 2 ? s : (s >> 1); }

// ------------------------------------------------------------------------------------------
// One ray (sv > 0 or < 0) of an item.  kdt: optical paths of the 2 x 2 nodes; sr: the three source rows
// of the previous plane (lower v row first); sc: source at the nodes; a_*: see the regimes below.
// REG 0: everything in the departure-carried part (a = 1); 1: all direct (a = 0); 2: general (a per row).
// SMALL: some optical path of the item is below DTAU_SERIES -> closed form and series are both evaluated
// and selected per band, branch-free.
template <int SU, int J, int REG, bool SMALL>
__device__ __forceinline__ f2 node_update(const f2 dt, const Row3& slo, const Row3& shi, const Row3& xlo, const Row3& xhi,
                                          const f2 sp, const float4 w, const float a_lo, const float a_hi, const float a_p)
{
    const f2 Xu = bil<SU, J>(xlo, xhi, w);
    const f2 t2 = mul2(dt, bc(-LOG2E));
    const f2 E = make_float2(ex2_approx(t2.x), ex2_approx(t2.y));
    f2 em1 = sub2(bc(1.f), E);                                     // 1 - e^-dt
    f2 wl = mul2(em1, make_float2(rcp_approx(dt.x), rcp_approx(dt.y)));   // (1 - e^-dt)/dt
    if (!SMALL && REG == 0) {
        const f2 d = bil_from<SU, J>(slo, shi, w, neg2(sp));       // S_u - S_p (weights sum to 1 exactly)
        f2 v = fma2(neg2(Xu), em1, Xu);                            // Xu * e^-dt
        return fma2(d, wl, v);
    }
    if (!SMALL && REG == 1) {
        const f2 pp = sub2(bc(1.f), wl);                           // psi_p = 1 - (1-E)/dt
        const f2 pu = sub2(em1, pp);                               // psi_u = (1 - E) - psi_p
        const f2 Su = bil<SU, J>(slo, shi, w);
        f2 v = fma2(neg2(Xu), em1, Xu);
        v = fma2(pu, Su, v);
        return fma2(pp, sp, v);
    }
    f2 pp = sub2(bc(1.f), wl);
    if (SMALL) {
        // series below DTAU_SERIES: psi_p directly (no cancellation), wl = 1 - psi_p, em1 = dt*wl
        const f2 nd = neg2(dt);
        f2 q = fma2(nd, bc(1.0f / 120.0f), bc(1.0f / 24.0f));
        q = fma2(nd, q, bc(1.0f / 6.0f));
        q = fma2(nd, q, bc(0.5f));
        const f2 pp2 = mul2(dt, q);
        const f2 wl2 = sub2(bc(1.f), pp2);
        const f2 e2 = mul2(dt, wl2);
        const bool sx = dt.x < DTAU_SERIES, sy = dt.y < DTAU_SERIES;
        pp = make_float2(sx ? pp2.x : pp.x, sy ? pp2.y : pp.y);
        wl = make_float2(sx ? wl2.x : wl.x, sy ? wl2.y : wl.y);
        em1 = make_float2(sx ? e2.x : em1.x, sy ? e2.y : em1.y);
    }
    const f2 pu = sub2(em1, pp);
    f2 v = fma2(neg2(Xu), em1, Xu);
    if (REG == 0) {
        const f2 d = bil_from<SU, J>(slo, shi, w, neg2(sp));
        return fma2(d, wl, v);
    } else if (REG == 1) {
        const f2 Su = bil<SU, J>(slo, shi, w);
        v = fma2(pu, Su, v);
        return fma2(pp, sp, v);
    } else {
        const f2 R0 = fma2(bc(w.y), sid<SU, J>(slo), mul2(bc(w.x), cen<J>(slo)));
        const f2 R1 = fma2(bc(w.w), sid<SU, J>(shi), mul2(bc(w.z), cen<J>(shi)));
        const f2 St = fma2(bc(a_hi), R1, mul2(bc(a_lo), R0));
        const f2 Sh = sub2(add2(R0, R1), St);
        const f2 Stp = mul2(bc(a_p), sp);
        v = fma2(sub2(St, Stp), wl, v);
        v = fma2(pu, Sh, v);
        return fma2(pp, sub2(sp, Stp), v);
    }
}

// exchange strips of a core item at a block end (out of line: one step in K)
__device__ __noinline__ void item_publish(const UnitDesc* __restrict__ Up, const int v0, const int u0, const int par_ex,
                                          const int s, const unsigned fl, const unsigned pos,
                                          const bool core0, const bool core1, const float4 o0, const float4 o1)
{
    const UnitDesc& U = *Up;
    const int rowN = (int)((pos >> 16) & 0xffu), c0 = 2 * (int)(pos >> 24);
    const int vN = v0 + rowN - HALO, ug = u0 + c0 - HALO;
    float* xe = U.Xex + 2 * ((((size_t)par_ex * NSLOT + s) * U.n_v + vN) * U.n_u2 + ug);
    if (core0 && (fl & IT_STRIP0)) __stcg(reinterpret_cast<float4*>(xe), o0);
    if (core1 && (fl & IT_STRIP1)) __stcg(reinterpret_cast<float4*>(xe + 2 * U.n_u2), o1);
}

// carried plane, seam histories and exchange strips of one ray of an item
template <int SU>
__device__ __forceinline__ void ray_store(const int s, const unsigned pos, const unsigned fl, const bool act0, const bool act1,
                                          const UnitDesc& U, const TileGeo& G, const StepCtx& C, const uint32_t aXw,
                                          const float4 o0, const float4 o1)
{
    const uint32_t BU8 = 8u * (uint32_t)G.BU;
    const uint32_t a_w = aXw + (uint32_t)xplane(U, s) * 8u * (uint32_t)G.BOXN + 8u * (pos & 0xffffu);
    const int c1 = (int)((fl >> IT_C1_SH) & 3u);
    if (c1 == 2) {
        if (act0) sts128(a_w, o0);
        if (act1) sts128(a_w + BU8, o1);
    } else {
        if (act0) sts64(a_w, make_float2(o0.x, o0.y));
        if (act1) sts64(a_w + BU8, make_float2(o1.x, o1.y));
    }
    const int rowN = (int)((pos >> 16) & 0xffu), c0 = 2 * (int)(pos >> 24);
    if (C.hist && (fl & IT_FARC)) {
        // far-u column of this ray: its values are the next pass's seam ghosts of this plane
        const bool second = (((SU < 0) ? G.dlo_u : G.dhi_u - 1) - c0) != 0;
        const f2 f0 = second ? make_float2(o0.z, o0.w) : make_float2(o0.x, o0.y);
        const f2 f1 = second ? make_float2(o1.z, o1.w) : make_float2(o1.x, o1.y);
        f2* g = C.Ghist + s * U.n_v + (G.v0 + rowN - HALO);
        if (act0 && (fl & IT_CORE0)) __stcg(g, f0);
        if (act1 && (fl & IT_CORE1)) __stcg(g + 1, f1);
    }
    if (C.hist && (fl & IT_SPECIAL)) {
        // far-v row of this ray (periodic v axis): the next pass's seam ghost row of this plane
        const bool svp = !(s & 2);
        const bool r1 = (rowN + 1 == (svp ? G.dhi_v - 1 : G.dlo_v));         // the far row is node row 1 (else row 0)
        const float4 fv = r1 ? o1 : o0;
        const bool okr = r1 ? (act1 && (fl & IT_CORE1)) : (act0 && (fl & IT_CORE0));
        f2* gv = C.Ghist + NSLOT * U.n_v + s * U.n_u2 + (G.u0 + c0 - HALO);
        if (okr) {
            if (c1 == 2) __stcg(reinterpret_cast<float4*>(gv), fv);
            else __stcg(gv, make_float2(fv.x, fv.y));
        }
    }
    if (C.strips && (fl & (IT_STRIP0 | IT_STRIP1)))
        item_publish(&U, G.v0, G.u0, C.par_ex, s, fl, pos, act0 && (fl & IT_CORE0), act1 && (fl & IT_CORE1), o0, o1);
}

__device__ __forceinline__ float4 scale4(const float f, const float4 a) { return make_float4(f * a.x, f * a.y, f * a.z, f * a.w); }
__device__ __forceinline__ float4 cat4(const f2 a, const f2 b) { return make_float4(a.x, a.y, b.x, b.y); }

// the 2 x 2 nodes of one ray.  R[0..2]: the three stencil rows (lower v first) of kaprho, S and X; node row i
// uses rows (i, i+1).
template <int SU, int REG, bool SMALL>
__device__ __forceinline__ void ray_rows(const f2 (&dt)[2][2], const Row3 (&sr)[3], const Row3 (&xr)[3], const float4 sc0, const float4 sc1,
                                         const float4 w, const float (&a)[3], const float ap0, const float ap1, float4& o0, float4& o1)
{
    const f2 v00 = node_update<SU, 0, REG, SMALL>(dt[0][0], sr[0], sr[1], xr[0], xr[1], make_float2(sc0.x, sc0.y), w, a[0], a[1], ap0);
    const f2 v01 = node_update<SU, 1, REG, SMALL>(dt[0][1], sr[0], sr[1], xr[0], xr[1], make_float2(sc0.z, sc0.w), w, a[0], a[1], ap0);
    const f2 v10 = node_update<SU, 0, REG, SMALL>(dt[1][0], sr[1], sr[2], xr[1], xr[2], make_float2(sc1.x, sc1.y), w, a[1], a[2], ap1);
    const f2 v11 = node_update<SU, 1, REG, SMALL>(dt[1][1], sr[1], sr[2], xr[1], xr[2], make_float2(sc1.z, sc1.w), w, a[1], a[2], ap1);
    o0 = cat4(v00, v01); o1 = cat4(v10, v11);
}

// ------------------------------------------------------------------------------------------
// One item: the 2 x 2 nodes of the (at most two) rays of one group.  aKp / aKc: previous / this plane
// (opacity box, source box one plane further); aXr / aXw: carried planes read / written this step.
template <int SU>
__device__ __forceinline__ void do_item(
    const unsigned pos, const unsigned flp, const unsigned flm, const UnitDesc& U, const TileGeo& G, const StepCtx& C,
    const uint32_t aKp, const uint32_t aKc, const uint32_t aXr, const uint32_t aXw)
{
    const int hj = C.hj;
    const bool dq_off = ((flp | flm) & IT_DQ) && hj == 0;
    const bool p0 = (int)((flp >> IT_D0_SH) & 7u) <= hj, p1 = (int)((flp >> IT_D1_SH) & 7u) <= hj;
    const bool m0 = (int)((flm >> IT_D0_SH) & 7u) <= hj, m1 = (int)((flm >> IT_D1_SH) & 7u) <= hj;
    const bool actp = (p0 || p1) && !dq_off, actm = (m0 || m1) && !dq_off;
    if (!(actp || actm)) return;
    const int sp_ = (SU < 0) ? 1 : 0, sm_ = sp_ + 2;            // slots of the two rays (sv > 0, sv < 0)
    const uint32_t BU8 = 8u * (uint32_t)G.BU, PLB = 8u * (uint32_t)G.BOXN;
    const uint32_t noff = 8u * (pos & 0xffffu);                  // node row 0, first node (bytes)
    const uint32_t a_c = aKc + noff;                             // this plane at the node rows
    const float4 sc0 = lds128(a_c + PLB);
    const float4 sc1 = lds128(a_c + PLB + BU8);
    float4 op0, op1, om0, om1;
    if (C.dplane) {
        const float fp = (U.ray[sp_].up ? 1.f : 0.f) - C.a_cur, fm = (U.ray[sm_].up ? 1.f : 0.f) - C.a_cur;
        op0 = scale4(fp, sc0); op1 = scale4(fp, sc1);
        om0 = scale4(fm, sc0); om1 = scale4(fm, sc1);
    } else {
        const uint32_t a_k = aKp + noff - BU8;                   // previous plane, row rowN - 1
        f2 dtp[2][2], dtm[2][2];
        float dmin = 3.0e38f;
        {
            Row3 kr[4];
            kr[1] = load_row<SU>(a_k + BU8);
            kr[2] = load_row<SU>(a_k + 2u * BU8);
            const float4 kc0 = lds128(a_c), kc1 = lds128(a_c + BU8);
            if (actp) {
                kr[0] = load_row<SU>(a_k);
                const float4 w = *reinterpret_cast<const float4*>(U.ray[sp_].w);
                const f2 kc = bc(U.ray[sp_].kc);
                dtp[0][0] = mul2(add2(make_float2(kc0.x, kc0.y), bil<SU, 0>(kr[0], kr[1], w)), kc);
                dtp[0][1] = mul2(add2(make_float2(kc0.z, kc0.w), bil<SU, 1>(kr[0], kr[1], w)), kc);
                dtp[1][0] = mul2(add2(make_float2(kc1.x, kc1.y), bil<SU, 0>(kr[1], kr[2], w)), kc);
                dtp[1][1] = mul2(add2(make_float2(kc1.z, kc1.w), bil<SU, 1>(kr[1], kr[2], w)), kc);
                dmin = fminf(min3(dtp[0][0].x, dtp[0][0].y, dtp[0][1].x), min3(dtp[0][1].y, dtp[1][0].x, dtp[1][0].y));
                dmin = min3(dmin, dtp[1][1].x, dtp[1][1].y);
            }
            if (actm) {
                kr[3] = load_row<SU>(a_k + 3u * BU8);
                const float4 w = *reinterpret_cast<const float4*>(U.ray[sm_].w);
                const f2 kc = bc(U.ray[sm_].kc);
                dtm[0][0] = mul2(add2(make_float2(kc0.x, kc0.y), bil<SU, 0>(kr[1], kr[2], w)), kc);
                dtm[0][1] = mul2(add2(make_float2(kc0.z, kc0.w), bil<SU, 1>(kr[1], kr[2], w)), kc);
                dtm[1][0] = mul2(add2(make_float2(kc1.x, kc1.y), bil<SU, 0>(kr[2], kr[3], w)), kc);
                dtm[1][1] = mul2(add2(make_float2(kc1.z, kc1.w), bil<SU, 1>(kr[2], kr[3], w)), kc);
                dmin = min3(dmin, min3(dtm[0][0].x, dtm[0][0].y, dtm[0][1].x), min3(dtm[0][1].y, dtm[1][0].x, dtm[1][0].y));
                dmin = min3(dmin, dtm[1][1].x, dtm[1][1].y);
            }
        }
        const bool small = dmin < DTAU_SERIES;
        Row3 sr[4];
        sr[1] = load_row<SU>(a_k + PLB + BU8);
        sr[2] = load_row<SU>(a_k + PLB + 2u * BU8);
        const int rowN = (int)((pos >> 16) & 0xffu);
#define RAY_BODY(REG, SM, DT, SR0, XR, W, A, P0, P1, O0, O1)                                                       \
        do { const Row3 srr[3] = {sr[SR0], sr[SR0 + 1], sr[SR0 + 2]};                                                \
             ray_rows<SU, REG, SM>(DT, srr, XR, sc0, sc1, W, A, P0, P1, O0, O1); } while (0)
#define RAY_DISPATCH(DT, SR0, XR, W, FL, SVP, O0, O1)                                                              \
        do {                                                                                                       \
            const int reg = G.zmarch ? C.zreg : (int)(((FL) >> IT_REG_SH) & 3u);                                    \
            const float one3[3] = {1.f, 1.f, 1.f}, zero3[3] = {0.f, 0.f, 0.f};                                     \
            if (reg == 0 && !small) RAY_BODY(0, false, DT, SR0, XR, W, one3, 1.f, 1.f, O0, O1);                    \
            else if (reg == 1 && !small) RAY_BODY(1, false, DT, SR0, XR, W, zero3, 0.f, 0.f, O0, O1);              \
            else {                                                                                                 \
                float a3[3], ap0, ap1;                                                                             \
                if (G.zmarch) { a3[0] = a3[1] = a3[2] = C.a_prev; ap0 = ap1 = C.a_cur; }                           \
                else {                                                                                             \
                    const int v0r = G.v0 + rowN - HALO - ((SVP) ? 1 : 0);                                          \
                    a3[0] = (v0r <= G.kstar) ? 1.f : 0.f;                                                          \
                    a3[1] = (v0r + 1 <= G.kstar) ? 1.f : 0.f;                                                      \
                    a3[2] = (v0r + 2 <= G.kstar) ? 1.f : 0.f;                                                      \
                    ap0 = (SVP) ? a3[1] : a3[0]; ap1 = (SVP) ? a3[2] : a3[1];                                      \
                }                                                                                                  \
                RAY_BODY(2, true, DT, SR0, XR, W, a3, ap0, ap1, O0, O1);                                           \
            }                                                                                                      \
        } while (0)
        if (actp) {
            sr[0] = load_row<SU>(a_k + PLB);
            const uint32_t a_x = aXr + (uint32_t)xplane(U, sp_) * PLB + noff - BU8;
            Row3 xr[3];
            xr[0] = load_row<SU>(a_x); xr[1] = load_row<SU>(a_x + BU8); xr[2] = load_row<SU>(a_x + 2u * BU8);
            const float4 w = *reinterpret_cast<const float4*>(U.ray[sp_].w);
            RAY_DISPATCH(dtp, 0, xr, w, flp, true, op0, op1);
            if (flp & (IT_DIR0 | IT_DIR1)) {
                // inflow row of a bounded v axis (v = z), upward ray: I = S on the bottom row
                const int vN = G.v0 + rowN - HALO;
                if (flp & IT_DIR0) op0 = scale4(1.f - ((vN <= G.kstar) ? 1.f : 0.f), sc0);
                if (flp & IT_DIR1) op1 = scale4(1.f - ((vN + 1 <= G.kstar) ? 1.f : 0.f), sc1);
            }
        }
        if (actm) {
            sr[3] = load_row<SU>(a_k + PLB + 3u * BU8);
            const uint32_t a_x = aXr + (uint32_t)xplane(U, sm_) * PLB + noff;
            Row3 xr[3];
            xr[0] = load_row<SU>(a_x); xr[1] = load_row<SU>(a_x + BU8); xr[2] = load_row<SU>(a_x + 2u * BU8);
            const float4 w = *reinterpret_cast<const float4*>(U.ray[sm_].w);
            RAY_DISPATCH(dtm, 1, xr, w, flm, false, om0, om1);
            if (flm & (IT_DIR0 | IT_DIR1)) {
                // downward ray: I = 0 on the top row
                const int vN = G.v0 + rowN - HALO;
                if (flm & IT_DIR0) om0 = scale4(0.f - ((vN <= G.kstar) ? 1.f : 0.f), sc0);
                if (flm & IT_DIR1) om1 = scale4(0.f - ((vN + 1 <= G.kstar) ? 1.f : 0.f), sc1);
            }
        }
#undef RAY_DISPATCH
#undef RAY_BODY
    }
    if (actp) ray_store<SU>(sp_, pos, flp, p0, p1, U, G, C, aXw, op0, op1);
    if (actm) ray_store<SU>(sm_, pos, flm, m0, m1, U, G, C, aXw, om0, om1);
}

// ------------------------------------------------------------------------------------------
// shared-memory carve-up of a CTA (float2 nodes), every part 128-byte aligned
struct SmemPlan {
    int BU, BV, BOXN, guardA, guardB, nitems, nghost_max, nhalo_max, nstage, nxp;
    __host__ __device__ SmemPlan(int WU, int WV, int ng, int nstage_) {
        nstage = nstage_; nxp = 2 * ng;
        BU = WU + 2 * HALO; BV = WV + 2 * HALO;
        BOXN = (BU * BV + 15) & ~15;
        guardA = 16;                                         // an item reads the node before its first row
        guardB = (2 * BU + 2 + 15) & ~15;                    // ... and up to two rows after its last
        // one group's items (pairs of node rows x node pairs; halo on the upwind u side and on both v sides), whole warps
        nitems = ((((WU + HALO) / 2) * ((WV + 2 * (KMAX - 1) + 1) / 2 + 1)) + 31) & ~31;
        nghost_max = NSLOT * (BU + BV);
        nhalo_max = NSLOT * ((WV + KMAX) * (HALO / 2) + KMAX * ((WU + HALO) / 2 + 1));
    }
    __host__ __device__ int nodes() const { return guardA + (nstage * 2 + 2 * nxp) * BOXN + guardB; }
    __host__ __device__ size_t bytes() const {
        return (size_t)nodes() * 8 + (size_t)nghost_max * sizeof(GhostEnt) + (size_t)nhalo_max * sizeof(HaloEnt);
    }
};

__device__ void run_task(TaskShared& S, const SweepMaps& maps, const int tile, f2* __restrict__ smf,
                         float* __restrict__ Qa, float* __restrict__ Qb, float* __restrict__ Itop_all,
                         int* abortf)
{
    const UnitDesc& U = S.U;
    const int tid = threadIdx.x, T = blockDim.x;
    const SmemPlan SP(U.WU, U.WV, U.ng, U.nstage);
    const int NST = U.nstage, NXP = SP.nxp;
    TileGeo G;
    const int tu = tile % U.ntu, tv = tile / U.ntu;
    G.u0 = tu * U.WU; G.v0 = tv * U.WV;
    G.wu = min(U.WU, U.n_u - G.u0); G.wv = min(U.WV, U.n_v - G.v0);
    G.BU = SP.BU; G.BV = SP.BV; G.BOXN = SP.BOXN;
    G.dlo_u = HALO - G.u0; G.dhi_u = HALO + U.n_u - G.u0;
    G.dlo_v = HALO - G.v0; G.dhi_v = HALO + U.n_v - G.v0;
    G.kstar = *U.kstar;
    const int mthick = (U.march == 2) ? U.mthick[2] : 0;     // z-march: planes below this level are optically thick
    G.zmarch = (U.march == 2);
    const int BU = G.BU, BV = G.BV, BOXN = G.BOXN;
    const int n_m = U.n_m, npass = U.npass, K = U.K;
    const int nsteps = n_m * npass;
    const bool zmarch = G.zmarch;
    const bool up_z = (U.dir > 0);                           // z-march: the unit's rays point up

    f2* const stage0 = smf + SP.guardA;                      // [NST][2][BOXN]
    f2* const Xb = stage0 + NST * 2 * BOXN;                  // [2][NXP][BOXN]
    GhostEnt* const gt = reinterpret_cast<GhostEnt*>(smf + SP.nodes());
    HaloEnt* const ht = reinterpret_cast<HaloEnt*>(gt + SP.nghost_max);
    uint64_t* const mbar = S.mbar;

    for (int i = tid; i < SP.nodes(); i += T) smf[i] = make_float2(0.f, 0.f);
    if (tid == 0) {
        for (int i = 0; i < NST; ++i) mbar_init(&mbar[i], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        S.flag = 0; S.nghost = 0; S.nhalo = 0;
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncthreads();

    // ---- coefficient planes through the TMA ring (started first: the tables below hide its latency)
    const CUtensorMap* const cmap = &maps.m[U.march];
    const uint32_t stage_bytes = 2u * (uint32_t)(BU * BV) * 8u;
    auto plane_of = [&](int mm) { return (U.dir > 0) ? mm : n_m - 1 - mm; };
    auto issue_load = [&](int pl, int st) {                  // one thread
        uint64_t* bar = &mbar[st];
        mbar_expect_tx(bar, stage_bytes);
        f2* dst = stage0 + (size_t)st * 2 * BOXN;
        const int c1 = zmarch ? G.v0 : (U.march == 1 ? pl + HALO : pl);
        const int c2 = zmarch ? pl : G.v0 - HALO;
        tensor_load4(dst, cmap, 2 * G.u0, c1, c2, 2 * U.pair, bar);
        tensor_load4(dst + BOXN, cmap, 2 * G.u0, c1, c2, 2 * U.pair + 1, bar);
    };
    if (tid == 0) {
        issue_load(plane_of(n_m - 1), NST - 1);              // the plane "before" step 0
        issue_load(plane_of(0), 0);
        if (nsteps > 1 && NST > 2) issue_load(plane_of(1 % n_m), 1);
    }

    // ---- the items of this thread.  The threads are split evenly between the unit's ray groups; item
    //      index e = tg + r * TG enumerates the 2 x 2 blocks of the group's region (tile core + upwind u halo
    //      + both v halos of depth K-1, clipped to the domain) row-pair by row-pair.
    const int TG = T / U.ng;
    const int grp = tid / TG, tg = tid - grp * TG;
    const int gsu = (U.ng == 2) ? (grp ? -1 : 1) : U.gsu0;    // su of this thread's group
    unsigned ipos[MAXIT], iflp[MAXIT], iflm[MAXIT];
    {
        const int hmax = K - 1;
        const int s_p = (gsu < 0) ? 1 : 0, s_m = s_p + 2;
        const bool on_p = U.ray[s_p].active != 0, on_m = U.ray[s_m].active != 0;
        const bool up_u = (gsu > 0) ? (tu > 0) : (tu < U.ntu - 1);
        const bool lo_v = (tv > 0), hi_v = (tv < U.ntv - 1);          // a tile below / above (upwind of sv > 0 / sv < 0)
        const int hu = (up_u && hmax > 0) ? HALO : 0;
        const int hvp = (lo_v && on_p) ? hmax : 0, hvm = (hi_v && on_m) ? hmax : 0;
        const int clo = max((gsu > 0) ? HALO - hu : HALO, G.dlo_u);
        const int chi = min((gsu > 0) ? HALO + G.wu : HALO + G.wu + hu, G.dhi_u);
        const int rlo = max(HALO - hvp, G.dlo_v);
        const int rhi = min(HALO + G.wv + hvm, G.dhi_v);
        const int qlo = clo >> 1, nq = ((chi + 1) >> 1) - qlo, np = (rhi - rlo + 1) >> 1;
#pragma unroll
        for (int r = 0; r < MAXIT; ++r) {
            const int e = tg + r * TG;
            unsigned pos = (unsigned)(HALO * BU + HALO) | ((unsigned)HALO << 16) | ((unsigned)(HALO / 2) << 24);
            unsigned fl2[2] = {IT_NEVER, IT_NEVER};
            if ((on_p || on_m) && rhi > rlo && chi > clo && e < nq * np) {
                const int pr = e / nq, q = qlo + (e - pr * nq);
                const int rowN = rlo + 2 * pr;
                pos = (unsigned)(rowN * BU + 2 * q) | ((unsigned)rowN << 16) | ((unsigned)q << 24);
                const int c0 = 2 * q;
                const bool core_q = (c0 >= HALO) && (c0 < HALO + G.wu);
                const int vN = G.v0 + rowN - HALO;
#pragma unroll
                for (int h = 0; h < 2; ++h) {                 // h = 0: ray sv > 0; 1: ray sv < 0
                    const bool svp = (h == 0);
                    if (!(svp ? on_p : on_m)) continue;
                    unsigned fl = 0;
                    auto depth = [&](int row) {
                        if (row < rlo || row >= rhi) return 7;
                        if (row < HALO) return svp ? HALO - row : 7;                   // below the core: halo of sv > 0 only
                        if (row >= HALO + G.wv) return svp ? 7 : row - (HALO + G.wv - 1);
                        return 0;
                    };
                    fl |= (unsigned)depth(rowN) << IT_D0_SH;
                    fl |= (unsigned)depth(rowN + 1) << IT_D1_SH;
                    if (!core_q) fl |= IT_DQ;
                    if (!zmarch) {
                        const int v0r = vN - (svp ? 1 : 0);
                        const unsigned reg = (v0r + 2 <= G.kstar) ? 0u : ((v0r > G.kstar) ? 1u : 2u);
                        fl |= reg << IT_REG_SH;
                        const int drow = svp ? 0 : U.n_v - 1;    // inflow row (x/y-march), global v
                        if (vN == drow) fl |= IT_DIR0;
                        if (vN + 1 == drow) fl |= IT_DIR1;
                    }
                    const bool c0r = core_q && rowN >= HALO && rowN < HALO + G.wv;
                    const bool c1r = core_q && rowN + 1 >= HALO && rowN + 1 < HALO + G.wv;
                    if (c0r) fl |= IT_CORE0;
                    if (c1r) fl |= IT_CORE1;
                    fl |= (unsigned)min(2, chi - c0) << IT_C1_SH;
                    const int fr = svp ? G.dhi_v - 1 : G.dlo_v;       // far-v row of this ray (box)
                    const int fc = (gsu > 0) ? G.dhi_u - 1 : G.dlo_u; // far-u column of this group (box)
                    const bool farc = (fc >= c0 && fc < c0 + 2);
                    const bool farr = U.per_v && ((c0r && rowN == fr) || (c1r && rowN + 1 == fr));
                    if ((c0r || c1r) && farc) fl |= IT_FARC;
                    if ((c0r || c1r) && farr) fl |= IT_SPECIAL;
                    const bool su_strip = (gsu > 0) ? (c0 + 2 > HALO + G.wu - K) : (c0 - HALO < K);
                    if (c0r && (su_strip || (svp ? (HALO + G.wv - 1 - rowN < K) : (rowN - HALO < K)))) fl |= IT_STRIP0;
                    if (c1r && (su_strip || (svp ? (HALO + G.wv - 2 - rowN < K) : (rowN + 1 - HALO < K)))) fl |= IT_STRIP1;
                    fl2[h] = fl;
                }
            }
            ipos[r] = pos; iflp[r] = fl2[0]; iflm[r] = fl2[1];
        }
    }
    // ---- seam ghosts of this tile (compact list)
    for (int e = tid; e < SP.nghost_max; e += T) {
        const int s = e / (BV + BU), i = e - s * (BV + BU);
        const int su = (s & 1) ? -1 : 1, sv = (s & 2) ? -1 : 1;
        if (!U.ray[s].active) continue;
        int xoff = -1, goff = 0, bvv = 0;
        const int gcol = (su > 0) ? G.dlo_u - 1 : G.dhi_u;
        const int grow = (sv > 0) ? G.dlo_v - 1 : G.dhi_v;
        if (i < BV) {                                        // ghost column, box row i
            int v = G.v0 - HALO + i;
            const bool okv = U.per_v || (v >= 0 && v < U.n_v);
            if (gcol >= 0 && gcol < BU && okv) { v = wrap(v, U.n_v); xoff = i * BU + gcol; goff = s * U.n_v + v; bvv = i; }
        } else if (U.per_v) {                                // ghost row, box column i - BV
            const int bu = i - BV;
            if (grow >= 0 && grow < BV) {
                const int u = wrap(G.u0 - HALO + bu, U.n_u);
                xoff = grow * BU + bu; goff = NSLOT * U.n_v + s * U.n_u2 + u; bvv = grow;
            }
        }
        if (xoff >= 0) {
            GhostEnt g; g.xoff = (unsigned short)xoff; g.bv = (unsigned short)bvv; g.goff = goff | (s << 28);
            gt[atomicAdd(&S.nghost, 1)] = g;
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
        const int clo = max((su > 0 && up_u) ? 0 : HALO, G.dlo_u);
        const int chi = min((su < 0 && up_u) ? HALO + G.wu + HALO : HALO + G.wu, G.dhi_u);
        const int q_lo = clo >> 1, nq = ((chi + 1) >> 1) - q_lo, nr = rhi - rlo;
        for (int e = tid; e < nr * nq; e += T) {
            const int r = e / nq, row = rlo + r, q = q_lo + (e - r * nq);
            const bool core = (row >= HALO && row < HALO + G.wv) && (2 * q >= HALO && 2 * q < HALO + G.wu);
            if (core) continue;
            HaloEnt h;
            h.xoff = (unsigned short)(row * BU + 2 * q); h.slot = (unsigned char)s;
            h.mask = (unsigned char)(max(0, clo - 2 * q) | (min(2, chi - 2 * q) << 4));
            h.goff = (G.v0 - HALO + row) * U.n_u2 + (G.u0 - HALO + 2 * q);
            ht[atomicAdd(&S.nhalo, 1)] = h;
        }
    }
    __syncthreads();
    const int ngh = S.nghost, nhalo = S.nhalo;

    auto wait_stage = [&](int st, uint32_t par, int code) {
        unsigned spins = 0;
        while (!mbar_try_wait(&mbar[st], par)) { if (spin_abort(abortf, spins, code)) break; }
    };
    auto a_of = [&](int level) { return (level <= G.kstar) ? 1.f : 0.f; };
    // value of I^(0) - a S at a box position of plane `msrc` (Sbox = its source-function box)
    auto x_initial = [&](const f2* Sbox, int s, int bv, int xo_in_box, int msrc) {
        const f2 Sv = Sbox[xo_in_box];
        float a; bool dn, up;
        if (zmarch) { a = a_of(plane_of(msrc)); dn = (msrc == 0); up = up_z; }
        else { const int v = G.v0 - HALO + bv; a = a_of(v); up = !(s & 2); dn = (v == (up ? 0 : U.n_v - 1)); }
        const float f = ((dn && !up) ? 0.f : 1.f) - a;
        return make_float2(f * Sv.x, f * Sv.y);
    };

    // ---- x/y-march: X^(0) on the plane before step 0, whole box (halo and ghosts included)
    wait_stage(NST - 1, 0u, 5);
    if (!zmarch) {
        const f2* Sp = stage0 + ((NST - 1) * 2 + 1) * BOXN;
        for (int i = tid; i < BU * BV; i += T) {
            const int bv = i / BU;
#pragma unroll
            for (int s = 0; s < NSLOT; ++s)
                if (U.ray[s].active) Xb[xplane(U, s) * BOXN + i] = x_initial(Sp, s, bv, i, n_m - 1);
        }
    }
    __syncthreads();

    float* const Qdst = U.q_in_B ? Qb : Qa;
    float* const Itop_b = Itop_all ? Itop_all + (long long)(2 * U.pair) * U.it_sb : nullptr;
    const size_t g_plane = (size_t)NSLOT * (U.n_v + U.n_u2);
    f2* const Gu2 = reinterpret_cast<f2*>(U.Gu);
    const f2* const Xex2 = reinterpret_cast<const f2*>(U.Xex);

    // heating and emergent intensity of a finished plane (last pass): reads the new carried
    // plane Xn and that plane's coefficients
    auto q_pass = [&](const f2* Kc, const f2* Xn, int m_done) {
        const f2* Sc = Kc + BOXN;
        const int pl = plane_of(m_done);
        const int nqc = (G.wu + 1) >> 1;
        const float qb1 = (U.nband_ok == 2) ? FOUR_PI : 0.f;
        for (int e = tid; e < nqc * G.wv; e += T) {
            const int row = e / nqc, q = e - row * nqc;
            const int bo = (HALO + row) * BU + HALO + 2 * q;
            const int v = G.v0 + row, u = G.u0 + 2 * q;
            const int nval = min(2, G.wu - 2 * q);
            const float4 kp = *reinterpret_cast<const float4*>(Kc + bo);
            const float4 sp = *reinterpret_cast<const float4*>(Sc + bo);
            const float a_p = zmarch ? a_of(pl) : a_of(v);
            const float shs = 1.0f - a_p;
            f2 acc0 = make_float2(0.f, 0.f), acc1 = make_float2(0.f, 0.f);    // node 0 / node 1, per band
            const f2 s0 = mul2(bc(shs), make_float2(sp.x, sp.y)), s1 = mul2(bc(shs), make_float2(sp.z, sp.w));
#pragma unroll
            for (int s = 0; s < NSLOT; ++s) {
                if (!U.ray[s].active) continue;
                const float4 x = *reinterpret_cast<const float4*>(Xn + xplane(U, s) * BOXN + bo);
                const float wq = U.ray[s].wq;
                acc0 = fma2(bc(wq), sub2(make_float2(x.x, x.y), s0), acc0);       // w_r (I - S)
                acc1 = fma2(bc(wq), sub2(make_float2(x.z, x.w), s1), acc1);
                if (Itop_b && U.ray[s].itop >= 0) {
                    const bool top = zmarch ? (m_done == n_m - 1 && up_z) : (v == U.nz - 1 && !(s & 2));
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
            float* qd = Qdst + (long long)pl * U.q_sm + (long long)v * U.q_sv + u;
            const float q0 = FOUR_PI * kp.x * acc0.x + qb1 * kp.y * acc0.y;
            const float q1 = FOUR_PI * kp.z * acc1.x + qb1 * kp.w * acc1.y;
            if (U.qvec && nval == 2) red_add2(qd, q0, q1);
            else { atomicAdd(qd, q0); if (nval == 2) atomicAdd(qd + 1, q1); }
        }
    };
    // halo of the carried plane at a block start: K-deep strips of the upwind neighbours' planes
    auto load_halos = [&](f2* Xc, int par) {
        const f2* xe0 = Xex2 + (size_t)par * NSLOT * (size_t)U.n_v * U.n_u2;
        for (int e = tid; e < nhalo; e += T) {
            const HaloEnt h = ht[e];
            const float4 x = __ldcg(reinterpret_cast<const float4*>(xe0 + (size_t)h.slot * U.n_v * U.n_u2 + h.goff));
            f2* d = Xc + xplane(U, h.slot) * BOXN + h.xoff;
            const int c0 = h.mask & 15, c1 = h.mask >> 4;
            if (c0 == 0 && c1 == 2) *reinterpret_cast<float4*>(d) = x;
            else if (c0 == 0) d[0] = make_float2(x.x, x.y);
            else if (c1 == 2) d[1] = make_float2(x.z, x.w);
        }
    };
    // seam ghosts: value of ghost entry g for the carried plane `msrc` from pass `psrc`
    auto ghost_fetch = [&](const GhostEnt g, int psrc, int msrc, const f2* Sbox) -> f2 {
        if (psrc < 0) return x_initial(Sbox, g.goff >> 28, g.bv, g.xoff, msrc);
        return __ldcg(Gu2 + ((size_t)(psrc & 1) * n_m + msrc) * g_plane + (g.goff & 0x0fffffff));
    };
    auto ghost_off = [&](const GhostEnt g) { return xplane(U, g.goff >> 28) * BOXN + g.xoff; };

    // ================================================================== the march
    int cur = 0, gblk = 0, s_ = 0;
    int stc = 0, stp = NST - 1;                              // stages of this step's and the previous plane
    uint32_t par_bits = 1u << (NST - 1);                     // stage NST-1 already served the plane before step 0
    bool bail = false;
    for (int pass = 0; pass < npass && !bail; ++pass) {
        const bool lastpass = (pass == npass - 1);
        for (int blk0 = 0; blk0 < n_m && !bail; blk0 += K) {
            const int blen = min(K, n_m - blk0);
            // ---- block start: wait for the unit, fetch halos and seam ghosts of the previous plane
            if (s_ > 0) {
                const bool exch = !(zmarch && blk0 == 0);
                const int m_prev = (blk0 == 0) ? n_m - 1 : blk0 - 1;
                // seam ghosts of the previous plane come from the previous pass: inside a pass (blk0 > 0)
                // they were written more than one block ago, i.e. before the arrival counter this tile
                // has already seen, so they are fetched before the wait and only stored after it (one
                // L2 round trip and one barrier less per block); at a pass start they belong to the
                // block the wait is for
                const bool pre = exch && pass > 0 && blk0 > 0 && ngh > 0;
                f2 gpre = make_float2(0.f, 0.f);
                if (pre && tid < ngh) gpre = ghost_fetch(gt[tid], pass - 1, m_prev, nullptr);
                if (tid == 0) {
                    const int need = gblk * U.ntiles;
                    const int ab = *reinterpret_cast<volatile int*>(abortf);
                    unsigned spins = 0, ns = 32;
                    while (ld_acquire(U.barrier) < need) {
                        if (spin_abort(abortf, spins, 3 | (s_ << 4))) { S.flag = 1; break; }
                        __nanosleep(ns);
                        if (ns < 2048) ns += ns;             // back off: a unit waiting for residency spins long
                    }
                    if (ab != 0) S.flag = 1;
                }
                __syncthreads();
                if (S.flag != 0) { bail = true; break; }     // uniform: the watchdog fired somewhere
                if (exch) {
                    // halo pairs lie inside the domain, ghost columns / rows outside it: disjoint stores
                    f2* const Xr = Xb + cur * NXP * BOXN;
                    load_halos(Xr, (gblk - 1) & 1);
                    if (ngh > 0) {
                        const f2* Sp = stage0 + (size_t)stp * 2 * BOXN + BOXN;
                        if (pre && tid < ngh) Xr[ghost_off(gt[tid])] = gpre;
                        for (int e = pre ? tid + T : tid; e < ngh; e += T) { const GhostEnt g = gt[e]; Xr[ghost_off(g)] = ghost_fetch(g, pass - 1, m_prev, Sp); }
                    }
                    __syncthreads();
                }
            }
            for (int j = 0; j < blen; ++j, ++s_) {
                const int m = blk0 + j;
                const int hj = blen - 1 - j;
                const bool blk_last = (hj == 0);
                const bool more = (s_ + 1 < nsteps);
                const int pl = plane_of(m);
                const f2* const Kp = stage0 + (size_t)stp * 2 * BOXN;
                const f2* const Kc = stage0 + (size_t)stc * 2 * BOXN;
                f2* const Xr = Xb + cur * NXP * BOXN;
                f2* const Xw = Xb + (cur ^ 1) * NXP * BOXN;

                wait_stage(stc, (par_bits >> stc) & 1u, 2 | (s_ << 4));
                par_bits ^= 1u << stc;
                // ---- heating / emergent intensity of the previous step's plane
                if (lastpass && m > 0) q_pass(Kp, Xr, m - 1);
                // ---- seam ghosts for the next step (previous pass, this plane): fetch now, store after the update
                const bool ghost_next = !blk_last && more && ngh > 0;
                f2 gval[2] = {make_float2(0.f, 0.f), make_float2(0.f, 0.f)};
                if (ghost_next && pass > 0) {
#pragma unroll
                    for (int i = 0; i < 2; ++i) { const int e = tid + i * T; if (e < ngh) gval[i] = ghost_fetch(gt[e], pass - 1, m, nullptr); }
                }

                // ---- the update
                StepCtx C;
                C.hj = hj; C.par_ex = gblk & 1;
                C.dplane = zmarch && (m == 0);
                C.hist = !lastpass;
                C.Ghist = Gu2 + ((size_t)(pass & 1) * n_m + m) * g_plane;
                C.strips = blk_last && more && !(zmarch && m == n_m - 1);
                C.a_prev = a_of(pl - U.dir); C.a_cur = a_of(pl);
                C.zreg = (C.a_prev != 0.f && C.a_cur != 0.f) ? 0 : ((C.a_prev == 0.f && C.a_cur == 0.f) ? 1 : 2);
                // Thick-plane shortcut (z-march, non-final passes): on planes pl <= mthick every optical path
                // exceeds DTAU_SKIP, e^-dtau is exactly 0 and the new plane does not depend on the carried one.
                // The planes pl < mthick only feed such planes (and seam ghosts that are multiplied by 0), so
                // their updates are skipped; plane mthick restarts from whatever finite values the buffers hold.
                if (!(zmarch && !lastpass && pl < mthick)) {
                    const uint32_t aKp = smem_u32(Kp), aKc = smem_u32(Kc), aXr = smem_u32(Xr), aXw = smem_u32(Xw);
#pragma unroll 1
                    for (int r = 0; r < MAXIT; ++r) {        // one copy of the item code per group sign
                        const unsigned pos_ = r ? ipos[1] : ipos[0], flp_ = r ? iflp[1] : iflp[0], flm_ = r ? iflm[1] : iflm[0];
                        if (gsu < 0) do_item<-1>(pos_, flp_, flm_, U, G, C, aKp, aKc, aXr, aXw);
                        else         do_item<+1>(pos_, flp_, flm_, U, G, C, aKp, aKc, aXr, aXw);
                    }
                }
                // ---- seam ghosts of this plane into the new carried plane
                if (ghost_next) {
                    if (pass > 0) {
#pragma unroll
                        for (int i = 0; i < 2; ++i) { const int e = tid + i * T; if (e < ngh) Xw[ghost_off(gt[e])] = gval[i]; }
                        for (int e = tid + 2 * T; e < ngh; e += T) { const GhostEnt g = gt[e]; Xw[ghost_off(g)] = ghost_fetch(g, pass - 1, m, nullptr); }
                    } else {
                        for (int e = tid; e < ngh; e += T) { const GhostEnt g = gt[e]; Xw[ghost_off(g)] = ghost_fetch(g, -1, m, Kc + BOXN); }
                    }
                }
                // ---- end of step; at a block end publish (release) before anybody waits
                __syncthreads();
                if (tid == 0) {
                    if (blk_last && more) { __threadfence(); atomicAdd(U.barrier, 1); }
                    const int ahead = NST - 1;               // planes in flight beyond the previous one
                    if (s_ + ahead < nsteps) {
                        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                        int m2 = m + ahead; if (m2 >= n_m) m2 %= n_m;
                        issue_load(plane_of(m2), stp);       // the previous plane's stage is free now
                    }
                }
                if (blk_last && more) ++gblk;
                cur ^= 1;
                stp = stc; stc = (stc + 1 == NST) ? 0 : stc + 1;
            }
        }
    }
    // heating / emergent intensity of the last plane
    if (!bail) q_pass(stage0 + (size_t)stp * 2 * BOXN, Xb + cur * NXP * BOXN, n_m - 1);
    __syncthreads();
    if (tid == 0)
        for (int i = 0; i < NST; ++i)
            asm volatile("mbarrier.inval.shared::cta.b64 [%0];" ::"r"(smem_u32(&mbar[i])) : "memory");
}

__global__ void __launch_bounds__(RTS_SWEEP_THREADS, 1)
rts_sweep_kernel(const __grid_constant__ SweepMaps maps, const UnitDesc* __restrict__ units, int nunits,
                 int total_tickets, int* ticket_counter,
                 float* __restrict__ Qa, float* __restrict__ Qb, float* __restrict__ Itop_all, int* abortf)
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
        run_task(S, maps, ticket - S.U.ticket_begin, reinterpret_cast<f2*>(smem_raw), Qa, Qb, Itop_all, abortf);
    }
}

}  // namespace rts
