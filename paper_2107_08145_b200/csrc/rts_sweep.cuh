// rts_sweep.cuh -- K_b, the persistent sweep kernel (stages B-E) for sm_100a.
//
// Work decomposition ("sweep kernel"):
//   unit  = (march axis, direction, band): the <= 4 rays (one per sign pair su, sv) whose
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
//   item  = a 4 x 2 node block of one ray: the thread-level unit of work.  Every thread owns the
//           same (at most two) items for the whole task; their descriptors live in registers.
//           The items of a slot (ray) fill whole warps, so the ray's signs are warp-uniform.
// Per step a CTA streams one (kaprho, S) plane box through a 3-stage TMA ring (one
// cp.async.bulk.tensor per field, completing on an mbarrier) and updates its items from
// registers and shared memory.
// Carried quantity: X = I - a*S with a = 1 at levels k <= kstar (optically thick part, where
// J - S would cancel) and a = 0 above (thin part, where I << S would cancel).
#pragma once
#include "rts_kernels.cuh"

#ifndef RTS_SWEEP_THREADS
#define RTS_SWEEP_THREADS 768   // most threads of a sweep CTA (<= 85 registers): one such CTA per SM, or two of half the size
#endif

#ifndef RTS_ONE_BODY
#define RTS_ONE_BODY 0
#endif

namespace rts {

struct SweepMaps { CUtensorMap m[3]; };

#ifdef RTS_TRACE
// phase clocks of the sweep (per warp, summed): tuning builds only
__device__ unsigned long long g_trace[16];
#define TR_DECL() unsigned tr_acc[8] = {0, 0, 0, 0, 0, 0, 0, 0}; long long tr_t0 = clock64()
#define TR_BEGIN() tr_t0 = clock64()
#define TR_MARK(i) do { const long long tr_t1 = clock64(); tr_acc[i] += (unsigned)(tr_t1 - tr_t0); tr_t0 = tr_t1; } while (0)
#define TR_FLUSH() do { if ((threadIdx.x & 31) == 0) for (int i_ = 0; i_ < 8; ++i_) atomicAdd(&g_trace[i_], (unsigned long long)tr_acc[i_]); } while (0)
#else
#define TR_DECL() do {} while (0)
#define TR_BEGIN() do {} while (0)
#define TR_MARK(i) do {} while (0)
#define TR_FLUSH() do {} while (0)
#endif      // coefficient tensor of the x-, y-, z-march units

// closed-form attenuation factors: em1 = 1 - e^-dt, wl = (1 - e^-dt)/dt
__device__ __forceinline__ void att_closed(float dt, float& em1, float& wl) {
    const float E = ex2_approx(-dt * LOG2E);
    em1 = 1.0f - E;
    wl = em1 * rcp_approx(dt);
}
// series below DTAU_SERIES: psi_p directly (no cancellation), wl = 1 - psi_p, em1 = dt*wl
__device__ __forceinline__ void att_series(float dt, float& em1, float& wl, float& pp) {
    pp = dt * (0.5f - dt * (1.0f / 6.0f - dt * (1.0f / 24.0f - dt * (1.0f / 120.0f))));
    wl = 1.0f - pp;
    em1 = dt * wl;
}

// 6 values of one box row around a quad: left neighbour, the quad, right neighbour
__device__ __forceinline__ void load_row6(const float* __restrict__ row, float (&o)[6])
{
    const float4 v = *reinterpret_cast<const float4*>(row);
    o[0] = row[-1]; o[1] = v.x; o[2] = v.y; o[3] = v.z; o[4] = v.w; o[5] = row[4];
}
// Loads / stores of the item code on 32-bit shared-window byte addresses: one add per row instead of
// an index add plus a generic-to-shared conversion per access.
__device__ __forceinline__ float4 lds128(const uint32_t a) {
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a));
    return v;
}
template <int OFF>
__device__ __forceinline__ float lds32(const uint32_t a) {
    float v;
    asm volatile("ld.shared.f32 %0, [%1+%2];" : "=f"(v) : "r"(a), "n"(OFF));
    return v;
}
__device__ __forceinline__ void sts128(const uint32_t a, const float4 v) {
    asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(a), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}
// the quad and the side column the ray looks at (SU > 0: left neighbour in o[0]; SU < 0: right in o[5])
template <int SU>
__device__ __forceinline__ void load_row5(const uint32_t row, float (&o)[6])
{
    const float4 v = lds128(row);
    o[1] = v.x; o[2] = v.y; o[3] = v.z; o[4] = v.w;
    if (SU > 0) { o[0] = lds32<-4>(row); o[5] = 0.f; }
    else        { o[5] = lds32<16>(row); o[0] = 0.f; }
}

// packed fp32 pairs (Blackwell FFMA2 / FMUL2): one issue slot for two nodes
__device__ __forceinline__ float2 fma2(const float2 a, const float2 b, const float2 c) {
    unsigned long long r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(*reinterpret_cast<const unsigned long long*>(&a)),
        "l"(*reinterpret_cast<const unsigned long long*>(&b)), "l"(*reinterpret_cast<const unsigned long long*>(&c)));
    return *reinterpret_cast<float2*>(&r);
}
__device__ __forceinline__ float2 mul2(const float2 a, const float2 b) {
    unsigned long long r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(*reinterpret_cast<const unsigned long long*>(&a)),
        "l"(*reinterpret_cast<const unsigned long long*>(&b)));
    return *reinterpret_cast<float2*>(&r);
}

// optical paths of one node row (4 nodes).  lo / hi: opacity of the previous plane on the two
// stencil rows (lower / higher v), kv = 0.5*ds * weights of (lo, lo side, hi, hi side).
template <int SU>
__device__ __forceinline__ void row_dtau(const float (&lo)[6], const float (&hi)[6], const float4 kp,
                                         const float4 kv, const float kc, float (&dt)[4])
{
    const float kpa[4] = {kp.x, kp.y, kp.z, kp.w};
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const int c = j + 1, cs = j + 1 - SU;
        dt[j] = kc * kpa[j] + kv.x * lo[c] + kv.y * lo[cs] + kv.z * hi[c] + kv.w * hi[cs];
    }
}

// update of one node row.  slo/shi: source function on the two stencil rows; xlo/xhi: carried
// quantity; wv: weights of (lo, lo side, hi, hi side).  REG 0: everything in the departure-carried
// part (a = 1); 1: all direct (a = 0); 2: mixed (a_lo, a_hi, a_p = a on the two rows and at the node).
// SMALL: some optical path of the item is below DTAU_SERIES -> both forms are evaluated and
// selected per node, branch-free (a branch inside the node loop would serialise the nodes).
template <int SU, int REG, bool SMALL>
__device__ __forceinline__ void row_update(
    const float (&dt)[4], const float (&slo)[6], const float (&shi)[6],
    const float (&xlo)[6], const float (&xhi)[6], const float4 spv,
    const float4 wv, const float a_lo, const float a_hi, const float a_p, float (&xp)[4])
{
    const float sp[4] = {spv.x, spv.y, spv.z, spv.w};
    if (REG != 2 && !SMALL) {
        // the common bodies: the bilinear sums per node (their side-column operands are not
        // pair-aligned), the attenuation factors and the final combination for two nodes per
        // instruction (fma.rn.f32x2); same operations, same order, same rounding as the scalar form
#pragma unroll
        for (int j = 0; j < 4; j += 2) {
            const int c = j + 1, cs = j + 1 - SU;
            const float2 Xu = make_float2(wv.x * xlo[c] + wv.y * xlo[cs] + wv.z * xhi[c] + wv.w * xhi[cs],
                                          wv.x * xlo[c + 1] + wv.y * xlo[cs + 1] + wv.z * xhi[c + 1] + wv.w * xhi[cs + 1]);
            const float2 dt2 = make_float2(dt[j], dt[j + 1]);
            const float2 t2 = mul2(dt2, make_float2(-LOG2E, -LOG2E));
            const float2 E2 = make_float2(ex2_approx(t2.x), ex2_approx(t2.y));
            const float2 em1 = fma2(E2, make_float2(-1.f, -1.f), make_float2(1.f, 1.f));
            const float2 wl = mul2(em1, make_float2(rcp_approx(dt2.x), rcp_approx(dt2.y)));
            float2 v = fma2(make_float2(-Xu.x, -Xu.y), em1, Xu);                  // Xu * e^-dt
            if (REG == 0) {
                float d0 = sp[j], d1 = sp[j + 1];
                d0 = fmaf(-wv.x, slo[c], d0); d0 = fmaf(-wv.y, slo[cs], d0); d0 = fmaf(-wv.z, shi[c], d0); d0 = fmaf(-wv.w, shi[cs], d0);
                d1 = fmaf(-wv.x, slo[c + 1], d1); d1 = fmaf(-wv.y, slo[cs + 1], d1); d1 = fmaf(-wv.z, shi[c + 1], d1); d1 = fmaf(-wv.w, shi[cs + 1], d1);
                v = fma2(make_float2(-d0, -d1), wl, v);
            } else {
                const float2 pp = fma2(wl, make_float2(-1.f, -1.f), make_float2(1.f, 1.f));   // psi_p = 1 - (1-E)/dt
                const float2 pu = fma2(pp, make_float2(-1.f, -1.f), em1);                    // psi_u = (1 - E) - psi_p
                float s0_ = wv.x * slo[c], s1_ = wv.x * slo[c + 1];
                s0_ = fmaf(wv.y, slo[cs], s0_); s0_ = fmaf(wv.z, shi[c], s0_); s0_ = fmaf(wv.w, shi[cs], s0_);
                s1_ = fmaf(wv.y, slo[cs + 1], s1_); s1_ = fmaf(wv.z, shi[c + 1], s1_); s1_ = fmaf(wv.w, shi[cs + 1], s1_);
                v = fma2(pu, make_float2(s0_, s1_), v);
                v = fma2(pp, make_float2(sp[j], sp[j + 1]), v);
            }
            xp[j] = v.x; xp[j + 1] = v.y;
        }
        return;
    }
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const int c = j + 1, cs = j + 1 - SU;
        const float Xu = wv.x * xlo[c] + wv.y * xlo[cs] + wv.z * xhi[c] + wv.w * xhi[cs];
        float em1, wl;
        att_closed(dt[j], em1, wl);
        float pp = 1.0f - wl;
        if (SMALL) {
            float e2, w2, pp2;
            att_series(dt[j], e2, w2, pp2);
            const bool sm = dt[j] < DTAU_SERIES;
            pp = sm ? pp2 : pp;
            em1 = sm ? e2 : em1;
            wl = sm ? w2 : wl;
        }
        float v = fmaf(-Xu, em1, Xu);                  // Xu * e^-dt
        if (REG == 0) {
            float dS = sp[j];
            dS = fmaf(-wv.x, slo[c], dS); dS = fmaf(-wv.y, slo[cs], dS);
            dS = fmaf(-wv.z, shi[c], dS); dS = fmaf(-wv.w, shi[cs], dS);
            v = fmaf(-dS, wl, v);
        } else if (REG == 1) {
            const float pu = em1 - pp;                 // psi_u = (1-E)/dt - E = (1 - E) - psi_p
            float Su = wv.x * slo[c];
            Su = fmaf(wv.y, slo[cs], Su); Su = fmaf(wv.z, shi[c], Su); Su = fmaf(wv.w, shi[cs], Su);
            v = fmaf(pu, Su, v);
            v = fmaf(pp, sp[j], v);
        } else {
            const float pu = em1 - pp;
            const float R0 = wv.x * slo[c] + wv.y * slo[cs];
            const float R1 = wv.z * shi[c] + wv.w * shi[cs];
            const float St = a_lo * R0 + a_hi * R1;
            const float Sh = (R0 + R1) - St;
            const float Stp = a_p * sp[j];
            v = fmaf(-(Stp - St), wl, v);
            v = fmaf(pu, Sh, v);
            v = fmaf(pp, sp[j] - Stp, v);
        }
        xp[j] = v;
    }
}

__device__ __forceinline__ void red_add4(float* p, const float a, const float b, const float c, const float d)
{
    asm volatile("red.relaxed.gpu.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
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


// Item descriptor (two registers, static for a task): pos = node offset in the box | first node
// row << 16 | quad << 24; fl = flags.  The item is the 4 x 2 node block (rows rowN, rowN+1;
// columns 4*quad ..) of one slot.
enum : unsigned {
    IT_SLOT = 3u,            // bits 0-1
    IT_D0_SH = 2,            // bits 2-4   halo depth of node row 0 (0: core side; 7: never active)
    IT_D1_SH = 5,            // bits 5-7   halo depth of node row 1
    IT_DQ = 1u << 8,         // halo quad: only active while the remaining halo depth is > 0
    IT_REG_SH = 11,          // bits 11-12 regime of the stencil rows (x/y-march; static)
    IT_DIR0 = 1u << 13,      // node row is the inflow row of a bounded v axis
    IT_DIR1 = 1u << 14,
    IT_CORE0 = 1u << 15,     // node row and quad belong to the tile core
    IT_CORE1 = 1u << 16,
    IT_C1_SH = 19,           // bits 19-21 one past the last valid column of the quad (1..4)
    IT_SPECIAL = 1u << 22,   // core item holding a far-v row of a periodic v axis: writes the seam history (in line)
    IT_FARC = 1u << 26,      // core item holding the far-u column of its ray: writes the seam history (in line)
    IT_STRIP0 = 1u << 23,    // core node row lies in an exchange strip
    IT_STRIP1 = 1u << 24
};
constexpr unsigned IT_NEVER = (7u << IT_D0_SH) | (7u << IT_D1_SH);
constexpr int MAXIT = 2;     // items per thread

struct GhostEnt { unsigned short xoff_lo, bv; int goff; };   // 8 bytes; slot = goff >> 28, xoff = xoff_lo + slot * BOXP

struct TaskShared {
    UnitDesc U;
    uint64_t mbar[NSTAGE];
    int ticket, flag, nghost, nhalo, pad0, pad1;
};

struct StepCtx {
    int m, pl, pass, hj, par_ex;       // plane counter, plane index, pass, remaining halo depth, exchange parity
    int zreg;                          // z-march: regime of this step (0, 1, 2)
    bool dplane;                       // z-march inflow plane: nodes are set, not updated
    bool hist, strips, lastpass;       // write seam histories / publish strips / reduce the heating this step
    float a_prev, a_cur;               // z-march: a on the previous / this plane
    float* Ghist;                      // seam history of this plane and pass (far columns, then far rows)
};

struct TileGeo {
    int u0, v0, wu, wv, BU, BV, BOXP;
    int dlo_u, dhi_u, dlo_v, dhi_v;    // domain bounds in box coordinates
    int kstar;
    bool zmarch;
};

// exchange strips of a core item at a block end (out of line: one step in K)
// core0 / core1: node row 0 / 1 is a core row and was updated this step
__device__ __noinline__ void item_publish(const UnitDesc* __restrict__ Up, const int v0, const int u0, const int par_ex,
                                          const unsigned fl, const unsigned pos,
                                          const bool core0, const bool core1, const float4 o0, const float4 o1)
{
    const UnitDesc& U = *Up;
    const int s = fl & IT_SLOT;
    const int rowN = (int)((pos >> 16) & 0xffu), cq0 = 4 * (int)(pos >> 24);
    const int vN = v0 + rowN - HALO, ug = u0 + cq0 - HALO;
    float* xe = U.Xex + (((size_t)par_ex * NSLOT + s) * U.n_v + vN) * U.n_u4 + ug;
    if (core0 && (fl & IT_STRIP0)) __stcg(reinterpret_cast<float4*>(xe), o0);
    if (core1 && (fl & IT_STRIP1)) __stcg(reinterpret_cast<float4*>(xe + U.n_u4), o1);
}

// ------------------------------------------------------------------------------------------
// One item (one ray, 4 x 2 nodes).  Kp / Kc: previous / this plane (opacity box, source box at +BOXP).
template <int SU>
__device__ __forceinline__ void do_item(
    const unsigned pos, const unsigned fl, const UnitDesc& U, const TileGeo& G, const StepCtx& C,
    const float* __restrict__ Kp, const float* __restrict__ Kc,
    const float* __restrict__ Xr_all, float* __restrict__ Xw_all)
{
    const int hj = C.hj;
    const bool act0 = (int)((fl >> IT_D0_SH) & 7u) <= hj;
    const bool act1 = (int)((fl >> IT_D1_SH) & 7u) <= hj;
    if (!(act0 || act1) || ((fl & IT_DQ) && hj == 0)) return;
    const int s = fl & IT_SLOT;
    const bool svp = !(s & 2);                               // sv > 0
    const uint32_t BU4 = 4u * (uint32_t)G.BU, BOXP4 = 4u * (uint32_t)G.BOXP;
    const uint32_t noff4 = 4u * (pos & 0xffffu);             // node row 0 (bytes)
    const uint32_t off4 = noff4 - (svp ? BU4 : 0u);          // first stencil row: rows (R0, R1, R2)
    const uint32_t a_c = smem_u32(Kc) + noff4;               // this plane at the node rows
    const float4 sc0 = lds128(a_c + BOXP4);
    const float4 sc1 = lds128(a_c + BOXP4 + BU4);
    float o0[4], o1[4];
    if (C.dplane) {
        const float f = (U.ray[s].up ? 1.f : 0.f) - C.a_cur;
        o0[0] = f * sc0.x; o0[1] = f * sc0.y; o0[2] = f * sc0.z; o0[3] = f * sc0.w;
        o1[0] = f * sc1.x; o1[1] = f * sc1.y; o1[2] = f * sc1.z; o1[3] = f * sc1.w;
    } else {
        float dt0[4], dt1[4];
        const uint32_t a_k0 = smem_u32(Kp) + off4, a_k1 = a_k0 + BU4, a_k2 = a_k1 + BU4;
        {
            float k0[6], k1[6], k2[6];
            load_row5<SU>(a_k0, k0);
            load_row5<SU>(a_k1, k1);
            load_row5<SU>(a_k2, k2);
            const float4 kv = *reinterpret_cast<const float4*>(U.ray[s].wk);
            const float kc = U.ray[s].kc;
            row_dtau<SU>(k0, k1, lds128(a_c), kv, kc, dt0);
            row_dtau<SU>(k1, k2, lds128(a_c + BU4), kv, kc, dt1);
        }
        bool small = false;
#pragma unroll
        for (int j = 0; j < 4; ++j) small |= (dt0[j] < DTAU_SERIES) | (dt1[j] < DTAU_SERIES);
        float s0[6], s1[6], s2[6], x0[6], x1[6], x2[6];
        {
            load_row5<SU>(a_k0 + BOXP4, s0);
            load_row5<SU>(a_k1 + BOXP4, s1);
            load_row5<SU>(a_k2 + BOXP4, s2);
            const uint32_t a_x0 = smem_u32(Xr_all) + (uint32_t)s * BOXP4 + off4;
            load_row5<SU>(a_x0, x0);
            load_row5<SU>(a_x0 + BU4, x1);
            load_row5<SU>(a_x0 + 2u * BU4, x2);
        }
        const float4 wv = *reinterpret_cast<const float4*>(U.ray[s].wx);
        const int reg = G.zmarch ? C.zreg : (int)((fl >> IT_REG_SH) & 3u);
#define ROWS2(REG, SM, A0, A1, A2, P0, P1)                                                  \
        do {                                                                                \
            row_update<SU, REG, SM>(dt0, s0, s1, x0, x1, sc0, wv, A0, A1, P0, o0);          \
            row_update<SU, REG, SM>(dt1, s1, s2, x1, x2, sc1, wv, A1, A2, P1, o1);          \
        } while (0)
        if (reg == 0) {
            if (small || RTS_ONE_BODY) ROWS2(0, true, 1.f, 1.f, 1.f, 1.f, 1.f); else ROWS2(0, false, 1.f, 1.f, 1.f, 1.f, 1.f);
        } else if (reg == 1) {
            if (small || RTS_ONE_BODY) ROWS2(1, true, 0.f, 0.f, 0.f, 0.f, 0.f); else ROWS2(1, false, 0.f, 0.f, 0.f, 0.f, 0.f);
        } else {
            // a on the three stencil rows and at the two node rows
            float a0, a1, a2, ap0, ap1;
            if (G.zmarch) { a0 = a1 = a2 = C.a_prev; ap0 = ap1 = C.a_cur; }
            else {
                const int v0r = G.v0 + (int)((pos >> 16) & 0xffu) - HALO - (svp ? 1 : 0);
                a0 = (v0r <= G.kstar) ? 1.f : 0.f;
                a1 = (v0r + 1 <= G.kstar) ? 1.f : 0.f;
                a2 = (v0r + 2 <= G.kstar) ? 1.f : 0.f;
                ap0 = svp ? a1 : a0; ap1 = svp ? a2 : a1;
            }
            ROWS2(2, true, a0, a1, a2, ap0, ap1);
        }
#undef ROWS2
        if (fl & (IT_DIR0 | IT_DIR1)) {
            // inflow row of a bounded v axis (v = z): I = S (upward, bottom row) or 0 (downward, top row)
            const int vN = G.v0 + (int)((pos >> 16) & 0xffu) - HALO;
            const float fu = svp ? 1.f : 0.f;
            if (fl & IT_DIR0) {
                const float f = fu - ((vN <= G.kstar) ? 1.f : 0.f);
                o0[0] = f * sc0.x; o0[1] = f * sc0.y; o0[2] = f * sc0.z; o0[3] = f * sc0.w;
            }
            if (fl & IT_DIR1) {
                const float f = fu - ((vN + 1 <= G.kstar) ? 1.f : 0.f);
                o1[0] = f * sc1.x; o1[1] = f * sc1.y; o1[2] = f * sc1.z; o1[3] = f * sc1.w;
            }
        }
    }

    // ---- carried plane for the next step
    const int c1 = (int)((fl >> IT_C1_SH) & 7u);
    const float4 v0_ = make_float4(o0[0], o0[1], o0[2], o0[3]), v1_ = make_float4(o1[0], o1[1], o1[2], o1[3]);
    if (c1 == 4) {
        const uint32_t a_w = smem_u32(Xw_all) + (uint32_t)s * BOXP4 + noff4;
        if (act0) sts128(a_w, v0_);
        if (act1) sts128(a_w + BU4, v1_);
    } else {
        float* xw = Xw_all + s * G.BOXP + (int)(pos & 0xffffu);
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            if (act0 && j < c1) xw[j] = o0[j];
            if (act1 && j < c1) xw[G.BU + j] = o1[j];
        }
    }
    if (C.hist && (fl & IT_FARC)) {
        // far-u column of this ray: its values are the next pass's seam ghosts of this plane
        const int rowN = (int)((pos >> 16) & 0xffu), fj = ((s & 1) ? G.dlo_u : G.dhi_u - 1) - 4 * (int)(pos >> 24);
        const float f0 = fj == 0 ? o0[0] : fj == 1 ? o0[1] : fj == 2 ? o0[2] : o0[3];
        const float f1 = fj == 0 ? o1[0] : fj == 1 ? o1[1] : fj == 2 ? o1[2] : o1[3];
        float* g = C.Ghist + s * U.n_v + (G.v0 + rowN - HALO);
        if (act0 && (fl & IT_CORE0)) __stcg(g, f0);
        if (act1 && (fl & IT_CORE1)) __stcg(g + 1, f1);
    }
    if (C.hist && (fl & IT_SPECIAL)) {
        // far-v row of this ray (periodic v axis): the next pass's seam ghost row of this plane
        const int rowN = (int)((pos >> 16) & 0xffu), cq0 = 4 * (int)(pos >> 24);
        const bool r1 = (rowN + 1 == (svp ? G.dhi_v - 1 : G.dlo_v));         // the far row is node row 1 (else row 0)
        const float4 fv = r1 ? v1_ : v0_;
        const bool okr = r1 ? (act1 && (fl & IT_CORE1)) : (act0 && (fl & IT_CORE0));
        float* gv = C.Ghist + NSLOT * U.n_v + s * U.n_u4 + (G.u0 + cq0 - HALO);
        const int nv_ = min(4, HALO + G.wu - cq0);
        if (okr) {
            if (nv_ == 4) __stcg(reinterpret_cast<float4*>(gv), fv);
            else { const float a[4] = {fv.x, fv.y, fv.z, fv.w}; for (int j = 0; j < nv_; ++j) __stcg(gv + j, a[j]); }
        }
    }
    if (C.strips && (fl & (IT_STRIP0 | IT_STRIP1)))
        item_publish(&U, G.v0, G.u0, C.par_ex, fl, pos, act0 && (fl & IT_CORE0), act1 && (fl & IT_CORE1), v0_, v1_);
}

// ------------------------------------------------------------------------------------------
// shared-memory carve-up of a CTA, every part 128-byte aligned
struct HaloEnt { unsigned short xoff_lo; unsigned char slot, mask; int goff; };   // mask = c0 | c1 << 4

struct SmemPlan {
    int BU, BV, BOXP, guardA, guardB, nitems, nghost_max, nhalo_max;
    __host__ __device__ SmemPlan(int WU, int WV) {
        BU = WU + 2 * HALO; BV = WV + 2 * HALO;
        BOXP = (BU * BV + 31) & ~31;
        guardA = (BU + 1 + 31) & ~31;                        // an item reads one row above / below its node rows
        guardB = (3 * BU + 4 + 31) & ~31;
        nitems = ((((WU + HALO) / 4) * ((WV + KMAX) / 2)) + 31) & ~31;   // one slot's items (largest region), whole warps
        nghost_max = NSLOT * (BU + BV);
        nhalo_max = NSLOT * (WV + KMAX + KMAX * ((WU + HALO) / 4));
    }
    __host__ __device__ int floats() const { return guardA + (NSTAGE * 2 + 2 * NSLOT) * BOXP + guardB; }
    __host__ __device__ size_t bytes() const {
        return (size_t)floats() * 4 + (size_t)nghost_max * sizeof(GhostEnt) + (size_t)nhalo_max * sizeof(HaloEnt);
    }
};

__device__ void run_task(TaskShared& S, const SweepMaps& maps, const int tile, float* __restrict__ smf,
                         float* __restrict__ Qa, float* __restrict__ Qb, float* __restrict__ Itop_all,
                         int* abortf)
{
    const UnitDesc& U = S.U;
    const int tid = threadIdx.x, T = blockDim.x;
    const SmemPlan SP(U.WU, U.WV);
    TileGeo G;
    const int tu = tile % U.ntu, tv = tile / U.ntu;
    G.u0 = tu * U.WU; G.v0 = tv * U.WV;
    G.wu = min(U.WU, U.n_u - G.u0); G.wv = min(U.WV, U.n_v - G.v0);
    G.BU = SP.BU; G.BV = SP.BV; G.BOXP = SP.BOXP;
    G.dlo_u = HALO - G.u0; G.dhi_u = HALO + U.n_u - G.u0;
    G.dlo_v = HALO - G.v0; G.dhi_v = HALO + U.n_v - G.v0;
    G.kstar = *U.kstar;
    const int mthick = (U.march == 2) ? *U.mthick : 0;   // z-march: planes below this level are optically thick
    G.zmarch = (U.march == 2);
    const int BU = G.BU, BV = G.BV, BOXP = G.BOXP;
    const int n_m = U.n_m, npass = U.npass, K = U.K;
    const int nsteps = n_m * npass;
    const bool zmarch = G.zmarch;
    const bool up_z = (U.dir > 0);                           // z-march: the unit's rays point up

    float* const stage0 = smf + SP.guardA;                   // [NSTAGE][2][BOXP]
    float* const Xb = stage0 + NSTAGE * 2 * BOXP;            // [2][NSLOT][BOXP]
    GhostEnt* const gt = reinterpret_cast<GhostEnt*>(smf + SP.floats());
    HaloEnt* const ht = reinterpret_cast<HaloEnt*>(gt + SP.nghost_max);
    uint64_t* const mbar = S.mbar;

    for (int i = tid; i < SP.floats(); i += T) smf[i] = 0.f;
    if (tid == 0) {
        for (int i = 0; i < NSTAGE; ++i) mbar_init(&mbar[i], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        S.flag = 0; S.nghost = 0; S.nhalo = 0;
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncthreads();

    // ---- coefficient planes through the TMA ring (started first: the tables below hide its latency)
    const CUtensorMap* const cmap = &maps.m[U.march];
    const uint32_t stage_bytes = 2u * (uint32_t)(BU * BV) * 4u;
    auto plane_of = [&](int mm) { return (U.dir > 0) ? mm : n_m - 1 - mm; };
    auto issue_load = [&](int pl, int st) {                  // one thread
        uint64_t* bar = &mbar[st];
        mbar_expect_tx(bar, stage_bytes);
        float* dst = stage0 + (size_t)st * 2 * BOXP;
        const int c1 = zmarch ? G.v0 : (U.march == 1 ? pl + HALO : pl);
        const int c2 = zmarch ? pl : G.v0 - HALO;
        tensor_load4(dst, cmap, G.u0, c1, c2, 2 * U.band, bar);
        tensor_load4(dst + BOXP, cmap, G.u0, c1, c2, 2 * U.band + 1, bar);
    };
    if (tid == 0) {
        issue_load(plane_of(n_m - 1), NSTAGE - 1);           // the plane "before" step 0
        issue_load(plane_of(0), 0);
        if (nsteps > 1) issue_load(plane_of(1 % n_m), 1);
    }

    // ---- the items of this thread.  Item index i = tid + r * T; slot = i / nitems (whole warps per
    //      slot), e = i % nitems enumerates the 4 x 2 blocks of the slot's region (tile core + upwind
    //      halo of depth K-1, clipped to the domain) row-pair by row-pair.
    unsigned ipos[MAXIT], ifl[MAXIT];
#pragma unroll
    for (int r = 0; r < MAXIT; ++r) {
        const int idx = tid + r * T;
        const int s = idx / SP.nitems, e = idx - s * SP.nitems;
        unsigned fl = IT_NEVER | (unsigned)(s & 3), pos = (unsigned)(HALO * BU + HALO) | ((unsigned)HALO << 16) | (1u << 24);
        if (s < NSLOT && U.ray[s].active) {
            const int hmax = K - 1;
            const int su = (s & 1) ? -1 : 1;
            const bool svp = !(s & 2);
            const bool up_u = (su > 0) ? (tu > 0) : (tu < U.ntu - 1);
            const bool up_v = svp ? (tv > 0) : (tv < U.ntv - 1);
            const int hu = (up_u && hmax > 0) ? HALO : 0, hv = up_v ? hmax : 0;
            const int clo = max((su > 0) ? HALO - hu : HALO, G.dlo_u);
            const int chi = min((su > 0) ? HALO + G.wu : HALO + G.wu + hu, G.dhi_u);
            const int rlo = max(svp ? HALO - hv : HALO, G.dlo_v);
            const int rhi = min(svp ? HALO + G.wv : HALO + G.wv + hv, G.dhi_v);
            const int qlo = clo >> 2, nq = ((chi + 3) >> 2) - qlo, np = (rhi - rlo + 1) >> 1;
            if (rhi > rlo && chi > clo && e < nq * np) {
                const int pr = e / nq, q = qlo + (e - pr * nq);
                const int rowN = rlo + 2 * pr;
                pos = (unsigned)(rowN * BU + 4 * q) | ((unsigned)rowN << 16) | ((unsigned)q << 24);
                fl = (unsigned)s;
                auto depth = [&](int row) {
                    if (row < rlo || row >= rhi) return 7;
                    return svp ? max(0, HALO - row) : max(0, row - (HALO + G.wv - 1));
                };
                fl |= (unsigned)depth(rowN) << IT_D0_SH;
                fl |= (unsigned)depth(rowN + 1) << IT_D1_SH;
                const int cq0 = 4 * q;
                const bool core_q = (cq0 >= HALO) && (cq0 < HALO + G.wu);
                if (!core_q) fl |= IT_DQ;
                const int vN = G.v0 + rowN - HALO;
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
                fl |= (unsigned)min(4, chi - cq0) << IT_C1_SH;
                const int fr = svp ? G.dhi_v - 1 : G.dlo_v;       // far-v row of this slot (box)
                const int fc = (su > 0) ? G.dhi_u - 1 : G.dlo_u;  // far-u column of this slot (box)
                const bool farc = (fc >= cq0 && fc < cq0 + 4);
                const bool farr = U.per_v && ((c0r && rowN == fr) || (c1r && rowN + 1 == fr));
                if ((c0r || c1r) && farc) fl |= IT_FARC;
                if ((c0r || c1r) && farr) fl |= IT_SPECIAL;
                const bool su_strip = (su > 0) ? (cq0 + 4 > HALO + G.wu - K) : (cq0 - HALO < K);
                if (c0r && (su_strip || (svp ? (HALO + G.wv - 1 - rowN < K) : (rowN - HALO < K)))) fl |= IT_STRIP0;
                if (c1r && (su_strip || (svp ? (HALO + G.wv - 2 - rowN < K) : (rowN + 1 - HALO < K)))) fl |= IT_STRIP1;
            }
        }
        ipos[r] = pos; ifl[r] = fl;
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
                xoff = grow * BU + bu; goff = NSLOT * U.n_v + s * U.n_u4 + u; bvv = grow;
            }
        }
        if (xoff >= 0) {
            GhostEnt g; g.xoff_lo = (unsigned short)xoff; g.bv = (unsigned short)bvv; g.goff = goff | (s << 28);
            gt[atomicAdd(&S.nghost, 1)] = g;
        }
    }
    // ---- halo quads fetched at a block start (depth K), compact list
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
        const int q_lo = clo >> 2, nq = ((chi + 3) >> 2) - q_lo, nr = rhi - rlo;
        for (int e = tid; e < nr * nq; e += T) {
            const int r = e / nq, row = rlo + r, q = q_lo + (e - r * nq);
            const bool core = (row >= HALO && row < HALO + G.wv) && (4 * q >= HALO && 4 * q < HALO + G.wu);
            if (core) continue;
            HaloEnt h;
            h.xoff_lo = (unsigned short)(row * BU + 4 * q); h.slot = (unsigned char)s;
            h.mask = (unsigned char)(max(0, clo - 4 * q) | (min(4, chi - 4 * q) << 4));
            h.goff = (G.v0 - HALO + row) * U.n_u4 + (G.u0 - HALO + 4 * q);
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
    auto x_initial = [&](const float* Sbox, int s, int bv, int xo_in_box, int msrc) {
        const float Sv = Sbox[xo_in_box];
        float a; bool dn, up;
        if (zmarch) { a = a_of(plane_of(msrc)); dn = (msrc == 0); up = up_z; }
        else { const int v = G.v0 - HALO + bv; a = a_of(v); up = !(s & 2); dn = (v == (up ? 0 : U.n_v - 1)); }
        return ((dn && !up) ? 0.f : Sv) - a * Sv;
    };

    // ---- x/y-march: X^(0) on the plane before step 0, whole box (halo and ghosts included)
    wait_stage(NSTAGE - 1, 0u, 5);
    if (!zmarch) {
        const float* Sp = stage0 + ((NSTAGE - 1) * 2 + 1) * BOXP;
        for (int i = tid; i < BU * BV; i += T) {
            const int bv = i / BU;
#pragma unroll
            for (int s = 0; s < NSLOT; ++s)
                if (U.ray[s].active) Xb[s * BOXP + i] = x_initial(Sp, s, bv, i, n_m - 1);
        }
    }
    __syncthreads();

    float* const Qdst = U.q_in_B ? Qb : Qa;
    float* const Itop_b = Itop_all ? Itop_all + (long long)U.band * U.it_sb : nullptr;
    const size_t g_plane = (size_t)NSLOT * (U.n_v + U.n_u4);

    // heating and emergent intensity of a finished plane (last pass): reads the new carried
    // plane Xn and that plane's coefficients
    auto q_pass = [&](const float* Kc, const float* Xn, int m_done) {
        const float* Sc = Kc + BOXP;
        const int pl = plane_of(m_done);
        const int nqc = (G.wu + 3) >> 2;
        for (int e = tid; e < nqc * G.wv; e += T) {
            const int row = e / nqc, q = e - row * nqc;
            const int bo = (HALO + row) * BU + HALO + 4 * q;
            const int v = G.v0 + row, u = G.u0 + 4 * q;
            const int nval = min(4, G.wu - 4 * q);
            const float4 kp = *reinterpret_cast<const float4*>(Kc + bo);
            const float4 sp = *reinterpret_cast<const float4*>(Sc + bo);
            const float a_p = zmarch ? a_of(pl) : a_of(v);
            const float shs = 1.0f - a_p;
            float acc[4] = {0.f, 0.f, 0.f, 0.f};
            const float spa[4] = {sp.x, sp.y, sp.z, sp.w};
#pragma unroll
            for (int s = 0; s < NSLOT; ++s) {
                if (!U.ray[s].active) continue;
                const float4 x = *reinterpret_cast<const float4*>(Xn + s * BOXP + bo);
                const float xa[4] = {x.x, x.y, x.z, x.w};
                const float wq = U.ray[s].wq;
#pragma unroll
                for (int j = 0; j < 4; ++j) acc[j] = fmaf(wq, xa[j] - shs * spa[j], acc[j]);   // w_r (I - S)
                if (Itop_b && U.ray[s].itop >= 0) {
                    const bool top = zmarch ? (m_done == n_m - 1 && up_z) : (v == U.nz - 1 && !(s & 2));
                    if (top) {
                        float* dst = Itop_b + (long long)U.ray[s].itop * U.it_sr + (zmarch ? (long long)v : (long long)pl) * U.it_so;
#pragma unroll
                        for (int j = 0; j < 4; ++j) if (j < nval) dst[(long long)(u + j) * U.it_su] = xa[j] + a_p * spa[j];
                    }
                }
            }
            float* qd = Qdst + (long long)pl * U.q_sm + (long long)v * U.q_sv + u;
            const float kpa[4] = {kp.x, kp.y, kp.z, kp.w};
#pragma unroll
            for (int j = 0; j < 4; ++j) acc[j] *= FOUR_PI * kpa[j];
            if (U.qvec && nval == 4) red_add4(qd, acc[0], acc[1], acc[2], acc[3]);   // one 16-byte reduction
            else {
#pragma unroll
                for (int j = 0; j < 4; ++j) if (j < nval) atomicAdd(qd + j, acc[j]);
            }
        }
    };
    // halo of the carried plane at a block start: K-deep strips of the upwind neighbours' planes
    auto load_halos = [&](float* Xc, int par) {
        const float* xe0 = U.Xex + (size_t)par * NSLOT * (size_t)U.n_v * U.n_u4;
        for (int e = tid; e < nhalo; e += T) {
            const HaloEnt h = ht[e];
            const float4 x = __ldcg(reinterpret_cast<const float4*>(xe0 + (size_t)h.slot * U.n_v * U.n_u4 + h.goff));
            float* d = Xc + h.slot * BOXP + h.xoff_lo;
            const int c0 = h.mask & 15, c1 = h.mask >> 4;
            if (c0 == 0 && c1 == 4) *reinterpret_cast<float4*>(d) = x;
            else { const float xa[4] = {x.x, x.y, x.z, x.w};
#pragma unroll
                   for (int j = 0; j < 4; ++j) if (j >= c0 && j < c1) d[j] = xa[j]; }
        }
    };
    // seam ghosts: value of ghost entry g for the carried plane `msrc` from pass `psrc`
    auto ghost_fetch = [&](const GhostEnt g, int psrc, int msrc, const float* Sbox) -> float {
        if (psrc < 0) return x_initial(Sbox, g.goff >> 28, g.bv, g.xoff_lo, msrc);
        return __ldcg(U.Gu + ((size_t)(psrc & 1) * n_m + msrc) * g_plane + (g.goff & 0x0fffffff));
    };
    auto ghost_off = [&](const GhostEnt g) { return (g.goff >> 28) * BOXP + g.xoff_lo; };

    // ================================================================== the march
    TR_DECL();
    int cur = 0, gblk = 0, s_ = 0;
    int stc = 0, stp = NSTAGE - 1;                           // stages of this step's and the previous plane
    uint32_t par_bits = 1u << (NSTAGE - 1);                  // stage NSTAGE-1 already served the plane before step 0
    bool bail = false;
    for (int pass = 0; pass < npass && !bail; ++pass) {
        const bool lastpass = (pass == npass - 1);
        for (int blk0 = 0; blk0 < n_m && !bail; blk0 += K) {
            const int blen = min(K, n_m - blk0);
            // ---- block start: wait for the unit, fetch halos and seam ghosts of the previous plane
            TR_BEGIN();
            if (s_ > 0) {
                const bool exch = !(zmarch && blk0 == 0);
                const int m_prev = (blk0 == 0) ? n_m - 1 : blk0 - 1;
                // seam ghosts of the previous plane come from the previous pass: inside a pass (blk0 > 0)
                // they were written more than one block ago, i.e. before the arrival counter this tile
                // has already seen, so they are fetched before the wait and only stored after it (one
                // L2 round trip and one barrier less per block); at a pass start they belong to the
                // block the wait is for
                const bool pre = exch && pass > 0 && blk0 > 0 && ngh > 0;
                float gpre = 0.f;
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
                TR_MARK(7);
                if (exch) {
                    // halo quads lie inside the domain, ghost columns / rows outside it: disjoint stores
                    float* const Xr = Xb + cur * NSLOT * BOXP;
                    load_halos(Xr, (gblk - 1) & 1);
                    if (ngh > 0) {
                        const float* Sp = stage0 + (size_t)stp * 2 * BOXP + BOXP;
                        if (pre && tid < ngh) Xr[ghost_off(gt[tid])] = gpre;
                        for (int e = pre ? tid + T : tid; e < ngh; e += T) { const GhostEnt g = gt[e]; Xr[ghost_off(g)] = ghost_fetch(g, pass - 1, m_prev, Sp); }
                    }
                    __syncthreads();
                }
            }
            TR_MARK(0);
            for (int j = 0; j < blen; ++j, ++s_) {
                const int m = blk0 + j;
                const int hj = blen - 1 - j;
                const bool blk_last = (hj == 0);
                const bool more = (s_ + 1 < nsteps);
                const int pl = plane_of(m);
                const float* const Kp = stage0 + (size_t)stp * 2 * BOXP;
                const float* const Kc = stage0 + (size_t)stc * 2 * BOXP;
                float* const Xr = Xb + cur * NSLOT * BOXP;
                float* const Xw = Xb + (cur ^ 1) * NSLOT * BOXP;

                wait_stage(stc, (par_bits >> stc) & 1u, 2 | (s_ << 4));
                par_bits ^= 1u << stc;
                TR_MARK(1);
                // ---- heating / emergent intensity of the previous step's plane
                if (lastpass && m > 0) q_pass(Kp, Xr, m - 1);
                // ---- seam ghosts for the next step (previous pass, this plane): fetch now, store after the update
                const bool ghost_next = !blk_last && more && ngh > 0;
                float gval[2] = {0.f, 0.f};
                if (ghost_next && pass > 0) {
#pragma unroll
                    for (int i = 0; i < 2; ++i) { const int e = tid + i * T; if (e < ngh) gval[i] = ghost_fetch(gt[e], pass - 1, m, nullptr); }
                }

                // ---- the update
                StepCtx C;
                C.m = m; C.pl = pl; C.pass = pass; C.hj = hj; C.par_ex = gblk & 1;
                C.dplane = zmarch && (m == 0);
                C.hist = !lastpass; C.lastpass = lastpass;
                C.Ghist = U.Gu + ((size_t)(pass & 1) * n_m + m) * g_plane;
                C.strips = blk_last && more && !(zmarch && m == n_m - 1);
                C.a_prev = a_of(pl - U.dir); C.a_cur = a_of(pl);
                C.zreg = (C.a_prev != 0.f && C.a_cur != 0.f) ? 0 : ((C.a_prev == 0.f && C.a_cur == 0.f) ? 1 : 2);
                TR_MARK(2);
                // Thick-plane shortcut (z-march, non-final passes): on planes pl <= mthick every optical path
                // exceeds DTAU_SKIP, e^-dtau is exactly 0 and the new plane does not depend on the carried one.
                // The planes pl < mthick only feed such planes (and seam ghosts that are multiplied by 0), so
                // their updates are skipped; plane mthick restarts from whatever finite values the buffers hold.
                if (!(zmarch && !lastpass && pl < mthick)) {
#pragma unroll 1
                    for (int r = 0; r < MAXIT; ++r) {        // one copy of the item code; the slot of an item is warp-uniform
                        const unsigned pos_ = r ? ipos[1] : ipos[0], fl_ = r ? ifl[1] : ifl[0];
                        if (fl_ & 1u) do_item<-1>(pos_, fl_, U, G, C, Kp, Kc, Xr, Xw);
                        else          do_item<+1>(pos_, fl_, U, G, C, Kp, Kc, Xr, Xw);
                    }
                }
                TR_MARK(3);
                // ---- seam ghosts of this plane into the new carried plane
                if (ghost_next) {
                    if (pass > 0) {
#pragma unroll
                        for (int i = 0; i < 2; ++i) { const int e = tid + i * T; if (e < ngh) Xw[ghost_off(gt[e])] = gval[i]; }
                        for (int e = tid + 2 * T; e < ngh; e += T) { const GhostEnt g = gt[e]; Xw[ghost_off(g)] = ghost_fetch(g, pass - 1, m, nullptr); }
                    } else {
                        for (int e = tid; e < ngh; e += T) { const GhostEnt g = gt[e]; Xw[ghost_off(g)] = ghost_fetch(g, -1, m, Kc + BOXP); }
                    }
                }
                // ---- end of step; at a block end publish (release) before anybody waits
                TR_MARK(4);
                __syncthreads();
                TR_MARK(5);
                if (tid == 0) {
                    if (blk_last && more) { __threadfence(); atomicAdd(U.barrier, 1); }
                    if (s_ + 2 < nsteps) {
                        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                        int m2 = m + 2; if (m2 >= n_m) m2 -= n_m; if (m2 >= n_m) m2 %= n_m;
                        issue_load(plane_of(m2), stp);       // the previous plane's stage is free now
                    }
                }
                TR_MARK(6);
                if (blk_last && more) ++gblk;
                cur ^= 1;
                stp = stc; stc = (stc + 1 == NSTAGE) ? 0 : stc + 1;
            }
        }
    }
    TR_FLUSH();
    // heating / emergent intensity of the last plane
    if (!bail) q_pass(stage0 + (size_t)stp * 2 * BOXP, Xb + cur * NSLOT * BOXP, n_m - 1);
    __syncthreads();
    if (tid == 0)
        for (int i = 0; i < NSTAGE; ++i)
            asm volatile("mbarrier.inval.shared::cta.b64 [%0];" ::"r"(smem_u32(&mbar[i])) : "memory");
}

#ifndef RTS_SWEEP_MINB
#define RTS_SWEEP_MINB 1
#endif
__global__ void __launch_bounds__(RTS_SWEEP_THREADS, RTS_SWEEP_MINB)
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
        run_task(S, maps, ticket - S.U.ticket_begin, reinterpret_cast<float*>(smem_raw), Qa, Qb, Itop_all, abortf);
    }
}

}  // namespace rts
