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
// Per step a CTA streams one (kaprho, S) plane box through a 3-stage TMA ring
// (cp.async.bulk rows completing on mbarriers) and updates, per thread, a 4 x 2 node block for
// all rays of the unit from registers (opacity / source neighbourhoods are shared by the rays).
// Carried quantity: X = I - a*S with a = 1 at levels k <= kstar (optically thick part, where
// J - S would cancel) and a = 0 above (thin part, where I << S would cancel).
#pragma once
#include "rts_kernels.cuh"

namespace rts {

struct GhostEnt { int xoff; int goff; int bv; int slot; };   // xoff < 0: unused

struct TaskShared {
    UnitDesc U;
    int4 reg[KMAX][NSLOT];     // per remaining halo depth hj: rows [x, y), cols [z, w) a slot updates (box coords)
    int4 uni[KMAX];            // union of the slots: first row (even), row pairs, first quad, quads
    uint64_t mbar[NSTAGE];
    int ticket, flag;
};

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

// 6 values of one box row around a quad: columns -1 .. 4 relative to the quad.  The centre
// float4 comes from shared memory; the side values come from the neighbouring lanes' float4 when
// those lanes hold the adjacent quads of the same row, else from shared memory.
__device__ __forceinline__ void load_row6(const float* __restrict__ row, bool l_ok, bool r_ok, float (&o)[6])
{
    const float4 v = *reinterpret_cast<const float4*>(row);
    float l = __shfl_up_sync(0xffffffffu, v.w, 1);
    float r = __shfl_down_sync(0xffffffffu, v.x, 1);
    if (!l_ok) l = row[-1];
    if (!r_ok) r = row[4];
    o[0] = l; o[1] = v.x; o[2] = v.y; o[3] = v.z; o[4] = v.w; o[5] = r;
}
// same, only the side the ray looks at (SU > 0: left); result in the 6-layout, other side unset
template <int SU>
__device__ __forceinline__ void load_row5(const float* __restrict__ row, bool l_ok, bool r_ok, float (&o)[6])
{
    const float4 v = *reinterpret_cast<const float4*>(row);
    o[1] = v.x; o[2] = v.y; o[3] = v.z; o[4] = v.w;
    if (SU > 0) {
        float l = __shfl_up_sync(0xffffffffu, v.w, 1);
        if (!l_ok) l = row[-1];
        o[0] = l; o[5] = 0.f;
    } else {
        float r = __shfl_down_sync(0xffffffffu, v.x, 1);
        if (!r_ok) r = row[4];
        o[5] = r; o[0] = 0.f;
    }
}

// optical paths of one node row (4 nodes) of a ray with u-sign SU
//   ko / ku : opacity of the previous plane on the node's own row / upwind row (6-layout)
template <int SU>
__device__ __forceinline__ void row_dtau(const float (&ko)[6], const float (&ku)[6], const float4 kp,
                                         const float4 kv, const float kc, float (&dt)[4])
{
    const float kpa[4] = {kp.x, kp.y, kp.z, kp.w};
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const int c = j + 1, cs = j + 1 - SU;
        dt[j] = kc * kpa[j] + kv.x * ko[c] + kv.y * ko[cs] + kv.z * ku[c] + kv.w * ku[cs];
    }
}

// update of one node row.  so/su_: source function on the own / upwind row; xo/xu: carried
// quantity.  REG 0: everything in the departure-carried part (a = 1); 1: all direct (a = 0);
// 2: mixed (a_o, a_u, a_p = a on the own row, the upwind row and at the node).
template <int SU, int REG>
__device__ __forceinline__ void row_update(
    const float (&dt)[4], const float (&so)[6], const float (&su_)[6],
    const float (&xo)[6], const float (&xu)[6], const float4 spv,
    const float4 wv, const float a_o, const float a_u, const float a_p, const bool any_small, float (&xp)[4])
{
    const float sp[4] = {spv.x, spv.y, spv.z, spv.w};
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const int c = j + 1, cs = j + 1 - SU;
        const float Xu = wv.x * xo[c] + wv.y * xo[cs] + wv.z * xu[c] + wv.w * xu[cs];
        float em1, wl;
        att_closed(dt[j], em1, wl);
        float pp = 1.0f - wl;
        if (any_small) {
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
            dS = fmaf(-wv.x, so[c], dS); dS = fmaf(-wv.y, so[cs], dS);
            dS = fmaf(-wv.z, su_[c], dS); dS = fmaf(-wv.w, su_[cs], dS);
            v = fmaf(-dS, wl, v);
        } else if (REG == 1) {
            const float pu = em1 - pp;                 // psi_u = (1-E)/dt - E = (1 - E) - psi_p
            float Su = wv.x * so[c];
            Su = fmaf(wv.y, so[cs], Su); Su = fmaf(wv.z, su_[c], Su); Su = fmaf(wv.w, su_[cs], Su);
            v = fmaf(pu, Su, v);
            v = fmaf(pp, sp[j], v);
        } else {
            const float pu = em1 - pp;
            const float R0 = wv.x * so[c] + wv.y * so[cs];
            const float R1 = wv.z * su_[c] + wv.w * su_[cs];
            const float St = a_o * R0 + a_u * R1;
            const float Sh = (R0 + R1) - St;
            const float Stp = a_p * sp[j];
            v = fmaf(-(Stp - St), wl, v);
            v = fmaf(pu, Sh, v);
            v = fmaf(pp, sp[j] - Stp, v);
        }
        xp[j] = v;
    }
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

// ------------------------------------------------------------------------------------------
// Everything a thread needs to finish one slot of its 4 x 2 block (stores, histories, strips).
struct StepCtx {
    int m, pl, pass, hj, par_ex;       // plane counter, plane index, pass, remaining halo depth, exchange parity
    bool dplane;                       // z-march inflow plane: nodes are set, not updated
    bool hist, strips;                 // write seam histories / publish strips this step
    float a_prev, a_cur;               // z-march: a on the previous / this plane
};

struct TileGeo {
    int u0, v0, wu, wv, BU, BV, BOX;
    int dlo_u, dhi_u, dlo_v, dhi_v;    // domain bounds in box coordinates
    int kstar;
    bool zmarch;
};

template <int SU, int SV>
__device__ __forceinline__ void do_slot(
    const int s, const TaskShared& S, const TileGeo& G, const StepCtx& C,
    const float* __restrict__ Xr, float* __restrict__ Xw,      // carried plane of this slot: read / write box
    const int boff, const int rowB, const int quad, const bool valid, const bool l_ok, const bool r_ok,
    const float (&dt)[2][4],
    const float (&sA)[6], const float (&sB)[6], const float (&sC)[6], const float (&sD)[6],
    const float4 scB, const float4 scC)
{
    const UnitDesc& U = S.U;
    const int4 rg = S.reg[C.hj][s];
    const bool actB = rowB >= rg.x && rowB < rg.y;
    const bool actC = rowB + 1 >= rg.x && rowB + 1 < rg.y;
    const int c0 = max(0, rg.z - 4 * quad), c1 = min(4, rg.w - 4 * quad);
    const bool act = valid && (c0 < c1) && (actB || actC);
    if (!__any_sync(0xffffffffu, act)) return;

    const int vB = G.v0 + rowB - HALO;                       // global v of node row B
    float o0[4], o1[4];
    if (C.dplane) {
        const float f = (U.ray[s].up ? 1.f : 0.f) - C.a_cur;
        o0[0] = f * scB.x; o0[1] = f * scB.y; o0[2] = f * scB.z; o0[3] = f * scB.w;
        o1[0] = f * scC.x; o1[1] = f * scC.y; o1[2] = f * scC.z; o1[3] = f * scC.w;
    } else {
        // carried plane: rows (A,B,C) for SV > 0, (B,C,D) for SV < 0
        float x0[6], x1[6], x2[6];
        const float* xr = Xr + boff + (SV > 0 ? -G.BU : 0);
        load_row5<SU>(xr, l_ok, r_ok, x0);
        load_row5<SU>(xr + G.BU, l_ok, r_ok, x1);
        load_row5<SU>(xr + 2 * G.BU, l_ok, r_ok, x2);
        bool small = false;
#pragma unroll
        for (int j = 0; j < 4; ++j) small |= (dt[0][j] < DTAU_SERIES) | (dt[1][j] < DTAU_SERIES);
        const bool any_small = __any_sync(0xffffffffu, act && small);
        const float4 wv = *reinterpret_cast<const float4*>(U.ray[s].wx);
        // regime of the three stencil rows
        int reg;
        float aA, aB, aC;                                    // a on rows (first, second, third) of this slot
        if (G.zmarch) {
            aA = aB = aC = C.a_prev;
            reg = (C.a_prev != 0.f && C.a_cur != 0.f) ? 0 : ((C.a_prev == 0.f && C.a_cur == 0.f) ? 1 : 2);
        } else {
            const int v1 = vB + (SV > 0 ? -1 : 0);           // global v of the slot's first row
            aA = (v1 <= G.kstar) ? 1.f : 0.f;
            aB = (v1 + 1 <= G.kstar) ? 1.f : 0.f;
            aC = (v1 + 2 <= G.kstar) ? 1.f : 0.f;
            reg = (aC != 0.f) ? 0 : ((aA == 0.f) ? 1 : 2);
        }
#define RTS_ROWS(REG)                                                                                  \
    if (SV > 0) {                                                                                      \
        row_update<SU, REG>(dt[0], sB, sA, x1, x0, scB, wv, aB, aA, G.zmarch ? C.a_cur : aB, any_small, o0); \
        row_update<SU, REG>(dt[1], sC, sB, x2, x1, scC, wv, aC, aB, G.zmarch ? C.a_cur : aC, any_small, o1); \
    } else {                                                                                           \
        row_update<SU, REG>(dt[0], sB, sC, x0, x1, scB, wv, aA, aB, G.zmarch ? C.a_cur : aA, any_small, o0); \
        row_update<SU, REG>(dt[1], sC, sD, x1, x2, scC, wv, aB, aC, G.zmarch ? C.a_cur : aB, any_small, o1); \
    }
        if (reg == 0) { RTS_ROWS(0) } else if (reg == 1) { RTS_ROWS(1) } else { RTS_ROWS(2) }
#undef RTS_ROWS
        if (!G.zmarch) {
            // inflow row of a bounded v axis (v = z): I = S (upward, bottom row) or 0 (downward, top row)
            const int drow = (SV > 0) ? 0 : U.n_v - 1;
            if (vB == drow) {
                const float f = (SV > 0 ? 1.f : 0.f) - ((vB <= G.kstar) ? 1.f : 0.f);
                o0[0] = f * scB.x; o0[1] = f * scB.y; o0[2] = f * scB.z; o0[3] = f * scB.w;
            }
            if (vB + 1 == drow) {
                const float f = (SV > 0 ? 1.f : 0.f) - ((vB + 1 <= G.kstar) ? 1.f : 0.f);
                o1[0] = f * scC.x; o1[1] = f * scC.y; o1[2] = f * scC.z; o1[3] = f * scC.w;
            }
        }
    }
    if (!act) return;

    // ---- carried plane for the next step
    float* xw = Xw + boff;
    const bool full = (c0 == 0) && (c1 == 4);
    if (actB) {
        if (full) *reinterpret_cast<float4*>(xw) = make_float4(o0[0], o0[1], o0[2], o0[3]);
        else { _Pragma("unroll") for (int j = 0; j < 4; ++j) if (j >= c0 && j < c1) xw[j] = o0[j]; }
    }
    if (actC) {
        if (full) *reinterpret_cast<float4*>(xw + G.BU) = make_float4(o1[0], o1[1], o1[2], o1[3]);
        else { _Pragma("unroll") for (int j = 0; j < 4; ++j) if (j >= c0 && j < c1) xw[G.BU + j] = o1[j]; }
    }
    if (!(C.hist || C.strips)) return;

    // ---- core nodes only from here on
    const int cq0 = 4 * quad;                                // box column of the quad
    const bool core_q = (cq0 >= HALO) && (cq0 < HALO + G.wu);
    const bool coreB = actB && rowB >= HALO && rowB < HALO + G.wv;
    const bool coreC = actC && rowB + 1 >= HALO && rowB + 1 < HALO + G.wv;
    if (!core_q || !(coreB || coreC)) return;
    const int ug = G.u0 + cq0 - HALO;                        // global u of the quad
    if (C.hist) {
        float* Gp = U.Gu + ((size_t)(C.pass & 1) * U.n_m + C.m) * (size_t)(NSLOT * (U.n_v + U.n_u4));
        // far-u column of this ray: u = n_u-1 (su > 0) or u = 0 (su < 0)
        const int fj = ((SU > 0) ? G.dhi_u - 1 : G.dlo_u) - cq0;
        if (fj >= 0 && fj < 4) {
            const float f0 = fj == 0 ? o0[0] : fj == 1 ? o0[1] : fj == 2 ? o0[2] : o0[3];
            const float f1 = fj == 0 ? o1[0] : fj == 1 ? o1[1] : fj == 2 ? o1[2] : o1[3];
            if (coreB) __stcg(Gp + s * U.n_v + vB, f0);
            if (coreC) __stcg(Gp + s * U.n_v + vB + 1, f1);
        }
        if (U.per_v) {
            const int fr = (SV > 0) ? G.dhi_v - 1 : G.dlo_v;  // far-v row (box)
            float* gv = Gp + NSLOT * U.n_v + s * U.n_u4 + ug;
            const int nv_ = min(4, HALO + G.wu - cq0);
            if (coreB && rowB == fr) {
                if (nv_ == 4) __stcg(reinterpret_cast<float4*>(gv), make_float4(o0[0], o0[1], o0[2], o0[3]));
                else { _Pragma("unroll") for (int j = 0; j < 4; ++j) if (j < nv_) __stcg(gv + j, o0[j]); }
            }
            if (coreC && rowB + 1 == fr) {
                if (nv_ == 4) __stcg(reinterpret_cast<float4*>(gv), make_float4(o1[0], o1[1], o1[2], o1[3]));
                else { _Pragma("unroll") for (int j = 0; j < 4; ++j) if (j < nv_) __stcg(gv + j, o1[j]); }
            }
        }
    }
    if (C.strips) {
        const bool su_strip = (SU > 0) ? (cq0 + 4 > HALO + G.wu - U.K) : (cq0 - HALO < U.K);
        float* xe = U.Xex + (((size_t)C.par_ex * NSLOT + s) * U.n_v + vB) * U.n_u4 + ug;
        if (coreB) {
            const bool sv_strip = (SV > 0) ? (HALO + G.wv - 1 - rowB < U.K) : (rowB - HALO < U.K);
            if (su_strip || sv_strip) __stcg(reinterpret_cast<float4*>(xe), make_float4(o0[0], o0[1], o0[2], o0[3]));
        }
        if (coreC) {
            const bool sv_strip = (SV > 0) ? (HALO + G.wv - 2 - rowB < U.K) : (rowB + 1 - HALO < U.K);
            if (su_strip || sv_strip) __stcg(reinterpret_cast<float4*>(xe + U.n_u4), make_float4(o1[0], o1[1], o1[2], o1[3]));
        }
    }
}

// ------------------------------------------------------------------------------------------
__device__ void run_task(TaskShared& S, const int tile, float* __restrict__ smf,
                         float* __restrict__ Qa, float* __restrict__ Qb, float* __restrict__ Itop_all,
                         int* abortf)
{
    const UnitDesc& U = S.U;
    const int tid = threadIdx.x, T = blockDim.x, lane = tid & 31;
    TileGeo G;
    const int tu = tile % U.ntu, tv = tile / U.ntu;
    G.u0 = tu * U.WU; G.v0 = tv * U.WV;
    G.wu = min(U.WU, U.n_u - G.u0); G.wv = min(U.WV, U.n_v - G.v0);
    G.BU = U.WU + 2 * HALO; G.BV = U.WV + 2 * HALO; G.BOX = G.BU * G.BV;
    G.dlo_u = HALO - G.u0; G.dhi_u = HALO + U.n_u - G.u0;
    G.dlo_v = HALO - G.v0; G.dhi_v = HALO + U.n_v - G.v0;
    G.kstar = *U.kstar;
    G.zmarch = (U.march == 2);
    const int BU = G.BU, BV = G.BV, BOX = G.BOX;
    const int n_m = U.n_m, npass = U.npass, K = U.K;
    const int nsteps = n_m * npass;
    const bool zmarch = G.zmarch;
    const bool up_z = (U.dir > 0);                           // z-march: the unit's rays point up

    // ---- shared memory: guard row | [NSTAGE][2][BOX] coefficient planes | [2][NSLOT][BOX] carried
    //      planes (double buffered) | guard row | ghost table
    float* const stage0 = smf + BU;
    float* const Xb = stage0 + NSTAGE * 2 * BOX;
    GhostEnt* const gt = reinterpret_cast<GhostEnt*>(Xb + 2 * NSLOT * BOX + BU);
    const int ngh = NSLOT * (BV + BU);
    uint64_t* const mbar = S.mbar;

    for (int i = tid; i < 2 * BU + (NSTAGE * 2 + 2 * NSLOT) * BOX; i += T) smf[i] = 0.f;
    if (tid == 0) {
        for (int i = 0; i < NSTAGE; ++i) mbar_init(&mbar[i], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        S.flag = 0;
    }
    // ---- regions per remaining halo depth (threads 0..15), ghost table (all threads)
    if (tid < KMAX * NSLOT) {
        const int hj = tid / NSLOT, s = tid % NSLOT;
        const int su = (s & 1) ? -1 : 1, sv = (s & 2) ? -1 : 1;
        int4 r = make_int4(0, 0, 0, 0);
        if (U.ray[s].active) {
            const bool up_u = (su > 0) ? (tu > 0) : (tu < U.ntu - 1);
            const bool up_v = (sv > 0) ? (tv > 0) : (tv < U.ntv - 1);
            const int hu = (up_u && hj > 0) ? HALO : 0, hv = up_v ? hj : 0;
            r.z = max((su > 0) ? HALO - hu : HALO, G.dlo_u);
            r.w = min((su > 0) ? HALO + G.wu : HALO + G.wu + hu, G.dhi_u);
            r.x = max((sv > 0) ? HALO - hv : HALO, G.dlo_v);
            r.y = min((sv > 0) ? HALO + G.wv : HALO + G.wv + hv, G.dhi_v);
        }
        S.reg[hj][s] = r;
    }
    for (int e = tid; e < ngh; e += T) {
        const int s = e / (BV + BU), i = e - s * (BV + BU);
        const int su = (s & 1) ? -1 : 1, sv = (s & 2) ? -1 : 1;
        GhostEnt g; g.xoff = -1; g.goff = 0; g.bv = 0; g.slot = s;
        if (U.ray[s].active) {
            const int gcol = (su > 0) ? G.dlo_u - 1 : G.dhi_u;
            const int grow = (sv > 0) ? G.dlo_v - 1 : G.dhi_v;
            if (i < BV) {                                    // ghost column, box row i
                int v = G.v0 - HALO + i;
                const bool okv = U.per_v || (v >= 0 && v < U.n_v);
                if (gcol >= 0 && gcol < BU && okv) {
                    v = wrap(v, U.n_v);
                    g.xoff = s * BOX + i * BU + gcol; g.goff = s * U.n_v + v; g.bv = i;
                }
            } else if (U.per_v) {                            // ghost row, box column i - BV
                const int bu = i - BV;
                if (grow >= 0 && grow < BV) {
                    const int u = wrap(G.u0 - HALO + bu, U.n_u);
                    g.xoff = s * BOX + grow * BU + bu; g.goff = NSLOT * U.n_v + s * U.n_u4 + u; g.bv = grow;
                }
            }
        }
        gt[e] = g;
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncthreads();
    if (tid < KMAX) {
        int rmin = 1 << 30, rmax = 0, cmin = 1 << 30, cmax = 0;
        for (int s = 0; s < NSLOT; ++s) {
            const int4 r = S.reg[tid][s];
            if (r.y > r.x && r.w > r.z) { rmin = min(rmin, r.x); rmax = max(rmax, r.y); cmin = min(cmin, r.z); cmax = max(cmax, r.w); }
        }
        int4 un = make_int4(0, 0, 0, 0);
        if (rmax > 0) { un.x = rmin & ~1; un.y = (rmax - un.x + 1) >> 1; un.z = cmin >> 2; un.w = ((cmax + 3) >> 2) - un.z; }
        S.uni[tid] = un;
    }

    // ---- coefficient box rows that exist in memory, copy width
    const int cr_lo = U.per_v ? 0 : max(0, G.dlo_v);
    const int cr_hi = U.per_v ? min(BV, U.n_v + 2 * HALO - G.v0) : min(BV, G.dhi_v);
    const int ncr = cr_hi - cr_lo;
    const int cbw = min(BU, U.P - G.u0);
    const uint32_t row_bytes = (uint32_t)cbw * 4u;
    const float* const csrc0 = U.cbase + U.c_off + (long long)(G.v0 - HALO) * U.c_v + G.u0;
    auto plane_of = [&](int mm) { return (U.dir > 0) ? mm : n_m - 1 - mm; };
    auto issue_load = [&](int pl, int st) {                  // warp 0, convergent
        uint64_t* bar = &mbar[st];
        if (lane == 0) mbar_expect_tx(bar, 2u * (uint32_t)ncr * row_bytes);
        __syncwarp();
        float* dst = stage0 + (size_t)st * 2 * BOX;
        const float* src = csrc0 + (long long)pl * U.c_m;
        for (int r = lane; r < 2 * ncr; r += 32) {
            const int f = (r >= ncr) ? 1 : 0, bv = cr_lo + r - f * ncr;
            bulk_load(dst + f * BOX + bv * BU, src + f * U.c_field + (long long)bv * U.c_v, row_bytes, bar);
        }
    };
    if (tid < 32) {
        issue_load(plane_of(n_m - 1), NSTAGE - 1);           // the plane "before" step 0
        issue_load(plane_of(0), 0);
        if (nsteps > 1) issue_load(plane_of(1 % n_m), 1);
    }
    __syncthreads();

    auto wait_stage = [&](int st, uint32_t par, int code) {
        unsigned spins = 0;
        while (!mbar_try_wait(&mbar[st], par)) { if (spin_abort(abortf, spins, code)) break; }
    };
    auto a_of = [&](int level) { return (level <= G.kstar) ? 1.f : 0.f; };
    // value of I^(0) - a S at a box position of plane `msrc` (stage Sbox = its source function)
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
        const float* Sp = stage0 + ((NSTAGE - 1) * 2 + 1) * BOX;
        for (int i = tid; i < BOX; i += T) {
            const int bv = i / BU;
#pragma unroll
            for (int s = 0; s < NSLOT; ++s)
                if (U.ray[s].active) Xb[s * BOX + i] = x_initial(Sp, s, bv, i, n_m - 1);
        }
    }
    __syncthreads();

    float* const Qdst = U.q_in_B ? Qb : Qa;
    float* const Itop_b = Itop_all ? Itop_all + (long long)U.band * U.it_sb : nullptr;
    const size_t g_plane = (size_t)NSLOT * (U.n_v + U.n_u4);

    // heating and emergent intensity of the plane finished in the previous step (last pass):
    // reads the new carried plane Xn and that plane's coefficients
    auto q_pass = [&](const float* Kc, const float* Sc, const float* Xn, int m_done) {
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
                const float4 x = *reinterpret_cast<const float4*>(Xn + s * BOX + bo);
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
            for (int j = 0; j < 4; ++j) if (j < nval) atomicAdd(qd + j, FOUR_PI * kpa[j] * acc[j]);
        }
    };

    // halo of the carried plane at a block start: K-deep strips of the upwind neighbours' planes
    auto load_halos = [&](float* Xc, int par) {
        for (int s = 0; s < NSLOT; ++s) {
            if (!U.ray[s].active) continue;
            const int su = (s & 1) ? -1 : 1, sv = (s & 2) ? -1 : 1;
            const bool up_u = (su > 0) ? (tu > 0) : (tu < U.ntu - 1);
            const bool up_v = (sv > 0) ? (tv > 0) : (tv < U.ntv - 1);
            // rows / columns of the halo-extended region (depth K), clipped to the domain
            const int rlo = max((sv > 0 && up_v) ? HALO - K : HALO, G.dlo_v);
            const int rhi = min((sv < 0 && up_v) ? HALO + G.wv + K : HALO + G.wv, G.dhi_v);
            const int clo = max((su > 0 && up_u) ? 0 : HALO, G.dlo_u);
            const int chi = min((su < 0 && up_u) ? HALO + G.wu + HALO : HALO + G.wu, G.dhi_u);
            const int q_lo = clo >> 2, q_hi = (chi + 3) >> 2, nq = q_hi - q_lo;
            const int nr = rhi - rlo;
            const float* xe = U.Xex + ((size_t)par * NSLOT + s) * (size_t)U.n_v * U.n_u4;
            for (int e = tid; e < nr * nq; e += T) {
                const int r = e / nq, row = rlo + r, q = q_lo + (e - r * nq);
                const bool core = (row >= HALO && row < HALO + G.wv) && (4 * q >= HALO && 4 * q < HALO + G.wu);
                if (core) continue;
                const int v = G.v0 - HALO + row, u = G.u0 - HALO + 4 * q;
                const float4 x = __ldcg(reinterpret_cast<const float4*>(xe + (size_t)v * U.n_u4 + u));
                float* d = Xc + s * BOX + row * BU + 4 * q;
                const int c0 = max(0, clo - 4 * q), c1 = min(4, chi - 4 * q);
                if (c0 == 0 && c1 == 4) *reinterpret_cast<float4*>(d) = x;
                else { const float xa[4] = {x.x, x.y, x.z, x.w};
#pragma unroll
                       for (int j = 0; j < 4; ++j) if (j >= c0 && j < c1) d[j] = xa[j]; }
            }
        }
    };
    // ghost columns / rows of the carried plane `msrc` (values of the previous pass `psrc`)
    auto ghost_fetch = [&](int e, int psrc, int msrc, const float* Sbox) -> float {
        const GhostEnt g = gt[e];
        if (g.xoff < 0) return 0.f;
        if (psrc < 0) return x_initial(Sbox, g.slot, g.bv, g.xoff - g.slot * BOX, msrc);
        return __ldcg(U.Gu + ((size_t)(psrc & 1) * n_m + msrc) * g_plane + g.goff);
    };
    auto ghost_store = [&](int e, float* Xc, float val) {
        const int xo = gt[e].xoff;
        if (xo >= 0) Xc[xo] = val;
    };

    // ================================================================== the march
    int m = 0, pass = 0, cur = 0, gblk = 0;
    for (int s_ = 0; s_ < nsteps; ++s_) {
        const int stc = s_ % NSTAGE, stp = (s_ + NSTAGE - 1) % NSTAGE;
        const uint32_t par_c = (uint32_t)((s_ / NSTAGE + (stc == NSTAGE - 1 ? 1 : 0)) & 1);
        const int blk0 = m - m % K, blen = min(K, n_m - blk0);
        const int hj = blen - 1 - (m - blk0);
        const bool blk_first = (m == blk0), blk_last = (hj == 0);
        const int pl = plane_of(m);
        const float* const Kp = stage0 + (size_t)stp * 2 * BOX;
        const float* const Sp = Kp + BOX;
        const float* const Kc = stage0 + (size_t)stc * 2 * BOX;
        const float* const Sc = Kc + BOX;
        float* const Xr = Xb + cur * NSLOT * BOX;
        float* const Xw = Xb + (cur ^ 1) * NSLOT * BOX;
        const int m_prev = (m == 0) ? n_m - 1 : m - 1;

        // ---- block start: wait for the unit, fetch halos and seam ghosts of the previous plane
        if (blk_first && s_ > 0) {
            if (tid == 0) {
                const int need = gblk * U.ntiles;
                const int ab = *reinterpret_cast<volatile int*>(abortf);
                unsigned spins = 0;
                while (ld_acquire(U.barrier) < need) {
                    if (spin_abort(abortf, spins, 3 | (s_ << 4))) { S.flag = 1; break; }
                    __nanosleep(64);
                }
                if (ab != 0) S.flag = 1;
            }
            __syncthreads();
            if (S.flag != 0) break;                          // uniform: the watchdog fired somewhere
            if (!(zmarch && m == 0)) {
                load_halos(Xr, (gblk - 1) & 1);
                __syncthreads();                             // halo quads may overlap a ghost column
                for (int e = tid; e < ngh; e += T) ghost_store(e, Xr, ghost_fetch(e, pass - 1, m_prev, Sp));
            }
            __syncthreads();
        }
        wait_stage(stc, par_c, 2 | (s_ << 4));
        const bool lastpass = (pass == npass - 1);
        // ---- heating / emergent intensity of the previous step's plane
        if (lastpass && m > 0) q_pass(Kp, Sp, Xr, m - 1);

        // ---- seam ghosts for the next step (previous pass, this plane): fetch now, store after the update
        const bool ghost_next = !blk_last && (s_ + 1 < nsteps);
        float gval[2] = {0.f, 0.f};
        if (ghost_next && pass > 0) {
#pragma unroll
            for (int i = 0; i < 2; ++i) { const int e = tid + i * T; if (e < ngh) gval[i] = ghost_fetch(e, pass - 1, m, Sc); }
        }

        // ---- the update: one 4 x 2 node block per thread and round, all slots
        StepCtx C;
        C.m = m; C.pl = pl; C.pass = pass; C.hj = hj; C.par_ex = gblk & 1;
        C.dplane = zmarch && (m == 0);
        C.hist = !lastpass;
        C.strips = blk_last && (s_ + 1 < nsteps) && !(zmarch && m == n_m - 1);
        C.a_prev = a_of(pl - U.dir); C.a_cur = a_of(pl);
        const int4 un = S.uni[hj];
        const int nitems = un.y * un.w;
        for (int it0 = 0; it0 < nitems; it0 += T) {
            const int it = it0 + tid;
            const bool valid = it < nitems;
            const int idx = min(it, nitems - 1);
            const int pr = idx / un.w, q = idx - pr * un.w;
            const int rowB = un.x + 2 * pr, quad = un.z + q;
            const int boff = rowB * BU + 4 * quad;
            const bool l_ok = (lane > 0) && (q > 0);
            const bool r_ok = (lane < 31) && (q < un.w - 1) && (it + 1 < nitems);
            float dt[NSLOT][2][4];
            float4 scB, scC;
            if (!C.dplane) {
                float kA[6], kB[6], kC[6], kD[6];
                load_row6(Kp + boff - BU, l_ok, r_ok, kA);
                load_row6(Kp + boff, l_ok, r_ok, kB);
                load_row6(Kp + boff + BU, l_ok, r_ok, kC);
                load_row6(Kp + boff + 2 * BU, l_ok, r_ok, kD);
                const float4 kcB = *reinterpret_cast<const float4*>(Kc + boff);
                const float4 kcC = *reinterpret_cast<const float4*>(Kc + boff + BU);
#define RTS_DT(s, SU, SV)                                                                       \
    if (U.ray[s].active) {                                                                      \
        const float4 kv = *reinterpret_cast<const float4*>(U.ray[s].wk);                        \
        const float kc = U.ray[s].kc;                                                           \
        row_dtau<SU>(kB, (SV > 0) ? kA : kC, kcB, kv, kc, dt[s][0]);                            \
        row_dtau<SU>(kC, (SV > 0) ? kB : kD, kcC, kv, kc, dt[s][1]);                            \
    }
                RTS_DT(0, +1, +1) RTS_DT(1, -1, +1) RTS_DT(2, +1, -1) RTS_DT(3, -1, -1)
#undef RTS_DT
            }
            float sA[6], sB[6], sC[6], sD[6];
            if (!C.dplane) {
                load_row6(Sp + boff - BU, l_ok, r_ok, sA);
                load_row6(Sp + boff, l_ok, r_ok, sB);
                load_row6(Sp + boff + BU, l_ok, r_ok, sC);
                load_row6(Sp + boff + 2 * BU, l_ok, r_ok, sD);
            }
            scB = *reinterpret_cast<const float4*>(Sc + boff);
            scC = *reinterpret_cast<const float4*>(Sc + boff + BU);
            if (U.ray[0].active) do_slot<+1, +1>(0, S, G, C, Xr, Xw, boff, rowB, quad, valid, l_ok, r_ok, dt[0], sA, sB, sC, sD, scB, scC);
            if (U.ray[1].active) do_slot<-1, +1>(1, S, G, C, Xr + BOX, Xw + BOX, boff, rowB, quad, valid, l_ok, r_ok, dt[1], sA, sB, sC, sD, scB, scC);
            if (U.ray[2].active) do_slot<+1, -1>(2, S, G, C, Xr + 2 * BOX, Xw + 2 * BOX, boff, rowB, quad, valid, l_ok, r_ok, dt[2], sA, sB, sC, sD, scB, scC);
            if (U.ray[3].active) do_slot<-1, -1>(3, S, G, C, Xr + 3 * BOX, Xw + 3 * BOX, boff, rowB, quad, valid, l_ok, r_ok, dt[3], sA, sB, sC, sD, scB, scC);
        }
        // ---- seam ghosts of this plane into the new carried plane
        if (ghost_next) {
            if (pass > 0) {
#pragma unroll
                for (int i = 0; i < 2; ++i) { const int e = tid + i * T; if (e < ngh) ghost_store(e, Xw, gval[i]); }
                for (int e = tid + 2 * T; e < ngh; e += T) ghost_store(e, Xw, ghost_fetch(e, pass - 1, m, Sc));
            } else {
                for (int e = tid; e < ngh; e += T) ghost_store(e, Xw, ghost_fetch(e, -1, m, Sc));
            }
        }
        // ---- end of step; at a block end publish (release) before anybody waits
        __syncthreads();
        if (blk_last && s_ + 1 < nsteps) {
            ++gblk;
            if (tid == 0) { __threadfence(); atomicAdd(U.barrier, 1); }
        }
        if (tid < 32 && s_ + 2 < nsteps) {
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            issue_load(plane_of((m + 2) % n_m), (s_ + 2) % NSTAGE);
        }
        cur ^= 1;
        if (++m == n_m) { m = 0; ++pass; }
    }
    // heating / emergent intensity of the last plane
    if (S.flag == 0) {
        const int sl = nsteps - 1;
        q_pass(stage0 + (size_t)(sl % NSTAGE) * 2 * BOX, stage0 + (size_t)(sl % NSTAGE) * 2 * BOX + BOX,
               Xb + cur * NSLOT * BOX, n_m - 1);
    }
    __syncthreads();
    if (tid == 0)
        for (int i = 0; i < NSTAGE; ++i)
            asm volatile("mbarrier.inval.shared::cta.b64 [%0];" ::"r"(smem_u32(&mbar[i])) : "memory");
}

__global__ void __launch_bounds__(256, 2)
rts_sweep_kernel(const UnitDesc* __restrict__ units, int nunits, int total_tickets, int* ticket_counter,
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
        run_task(S, ticket - S.U.ticket_begin, reinterpret_cast<float*>(smem_raw), Qa, Qb, Itop_all, abortf);
    }
}

}  // namespace rts
