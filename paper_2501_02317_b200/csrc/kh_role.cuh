// kh_role.cuh -- KRATOS_KERNEL_ROLES: the fused Heun-stage kernel of the mixed-precision 3D path
// (float_t = fp32, float2_t = fp64), warp-specialised.
//
// The paired kernel (kh_pair.cuh) is bound by latency, not by HBM or by a pipe: its main warps need
// ~184 registers, so only two of them fit per scheduler and every dependent-issue gap shows
// (profiles/r1c).  Here the same work, on the same 32 x 16 tile with two cells per thread and packed
// f32x2 arithmetic, is split over three kinds of warps that each keep a small state, so that twenty
// warps share the SM and cover each other's latencies:
//
//   ZU warps (8)   own the columns of the tile along z: fetch the fp64 state (cp.async ring), recover the
//                  primitives (Sec. 3.1), publish them as the plane's tile, march the z
//                  slopes (Eq. 3) and z-face HLLC fluxes (Eq. 4-5) in registers, and do the fp64
//                  flux-difference update and Heun average plus the CFL rate of
//                  the new state;
//   XY warps (8)   do nothing but the in-plane Riemann problems: x / y slopes from the tile, left states
//                  exchanged through shared memory, HLLC at the low x face and the two low y faces of
//                  their cell pair, fluxes published in float_t;
//   halo warps (4) load and recover the 2-cell halo ring (boundary rules of Sec. 3.1.1 applied on load,
//                  PAPER.md:177-187), limit the cells next to the tile and solve the faces on the tile's
//                  two high edges.
//
// The roles hand tiles and fluxes to one another through double-buffered shared memory guarded by named
// barriers (bar.arrive by the producer, bar.sync by the consumer), so ZU works on plane k+1/k+2 while XY
// solves plane k; the only all-hands barrier left is the one between XY's slope and flux phases.
//
// Every flux is converted to float2_t by the ZU thread that applies it, from the one float_t value the
// solving thread published: both cells of a face add and subtract the very same number, so the totals are
// conserved to float2_t accuracy.  A face on a tile seam is solved by two thread blocks
// (edge solve of one, own face of the other) with one and the same sequence of explicitly rounded
// operations (hllcv below serves float and float2 alike), so both get the same bits.
#pragma once
#include <cuda_pipeline_primitives.h>

#include "kh_device.cuh"
#include "kh_pair.cuh"

namespace kh {
namespace rl {

using pr::f2;
using pr::Gas;
using pr::PRP;
using pr::PTX;
using pr::PTY;

constexpr int NW_ZU = PRP, NW_XY = PRP, NW_HALO = 4;
constexpr int WARP_XY0 = NW_ZU, WARP_H0 = NW_ZU + NW_XY;
constexpr int NWARPS = NW_ZU + NW_XY + NW_HALO;
constexpr int NTHREADS = NWARPS * 32;  // 640
constexpr int NRAW = 4;                // raw ring depth: fetched at plane s+3, recovered at s+2, updated at s
// registers: the block's pool is what it was launched with, 640 threads x 96; the halo group gives 32 per
// thread back and the four main groups take 8 each (640*96 = 512*104 + 128*64)
#define KH_ROLE_MAIN_REGS "104"
#define KH_ROLE_HALO_REGS "64"

// named barriers (0 is __syncthreads)
enum : int { BAR_AB = 1, BAR_WT_FULL = 2, BAR_WT_FREE = 4, BAR_F_FULL = 6, BAR_F_FREE = 8 };
constexpr int CNT_AB = (NW_XY + NW_HALO) * 32;
constexpr int CNT_ALL = NTHREADS;

__device__ __forceinline__ void bar_sync(int id, int count)
{
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(count) : "memory");
}
__device__ __forceinline__ void bar_arrive(int id, int count)
{
    asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(count) : "memory");
}

// ---- one source for scalar and packed arithmetic (explicitly rounded, see kh_device.cuh) ----------
struct P2 { bool x, y; };
__device__ __forceinline__ float vadd(float a, float b) { return __fadd_rn(a, b); }
__device__ __forceinline__ float vsub(float a, float b) { return __fadd_rn(a, -b); }
__device__ __forceinline__ float vmul(float a, float b) { return __fmul_rn(a, b); }
__device__ __forceinline__ float vfma(float a, float b, float c) { return __fmaf_rn(a, b, c); }
__device__ __forceinline__ float vneg(float a) { return -a; }
__device__ __forceinline__ float vmaxs(float a, float s) { return fmaxf(a, s); }
__device__ __forceinline__ float vrcp(float a) { return rcp_(a); }
__device__ __forceinline__ float vsqrt(float a) { return sqrt_(a); }
__device__ __forceinline__ float vrsqrt(float a) { return rsqrt_(a); }
__device__ __forceinline__ bool vge0(float a) { return a >= 0.0f; }
__device__ __forceinline__ bool vle0(float a) { return a <= 0.0f; }
__device__ __forceinline__ bool vor(bool a, bool b) { return a || b; }
__device__ __forceinline__ float vsel(bool c, float a, float b) { return c ? a : b; }
__device__ __forceinline__ void vset(float& v, float s) { v = s; }

__device__ __forceinline__ f2 vadd(f2 a, f2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ f2 vsub(f2 a, f2 b) { return __fadd2_rn(a, make_float2(-b.x, -b.y)); }
__device__ __forceinline__ f2 vmul(f2 a, f2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ f2 vfma(f2 a, f2 b, f2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ f2 vneg(f2 a) { return make_float2(-a.x, -a.y); }
__device__ __forceinline__ f2 vmaxs(f2 a, float s) { return make_float2(fmaxf(a.x, s), fmaxf(a.y, s)); }
__device__ __forceinline__ f2 vrcp(f2 a) { return make_float2(rcp_(a.x), rcp_(a.y)); }
__device__ __forceinline__ f2 vsqrt(f2 a) { return make_float2(sqrt_(a.x), sqrt_(a.y)); }
__device__ __forceinline__ f2 vrsqrt(f2 a) { return make_float2(rsqrt_(a.x), rsqrt_(a.y)); }
__device__ __forceinline__ P2 vge0(f2 a) { return P2{a.x >= 0.0f, a.y >= 0.0f}; }
__device__ __forceinline__ P2 vle0(f2 a) { return P2{a.x <= 0.0f, a.y <= 0.0f}; }
__device__ __forceinline__ P2 vor(P2 a, P2 b) { return P2{a.x || b.x, a.y || b.y}; }
__device__ __forceinline__ f2 vsel(P2 c, f2 a, f2 b) { return make_float2(c.x ? a.x : b.x, c.y ? a.y : b.y); }
__device__ __forceinline__ void vset(f2& v, float s) { v = make_float2(s, s); }

template <class V>
__device__ __forceinline__ V vbc(float s)
{
    V v;
    vset(v, s);
    return v;
}

// Face states of a cell from its value and its two neighbours (Eq. 3, reading S8):
// qL = q + minmod(q - qm, qp - q)/2 (left state of the high face), qR = q - minmod(...)/2.
__device__ __forceinline__ void vplm(float qm, float q, float qp, float& qL, float& qR)
{
    const float s = minmod(vsub(q, qm), vsub(qp, q));
    qL = vfma(0.5f, s, q);
    qR = vfma(-0.5f, s, q);
}
__device__ __forceinline__ void vplm(f2 qm, f2 q, f2 qp, f2& qL, f2& qR) { pr::plm(qm, q, qp, qL, qR); }

// Sec. 3.2.2: HLLC with the wave speeds of Eq. 5 and the contact speed of Eq. 4.
// Same formulas and order of operations as kh::hllc (kh_device.cuh), where they are documented; states are
// (rho, p - pref, u, v, w) with u normal to the face; result (mass, normal momentum - pref, tangential 1,
// tangential 2, energy).  V = float (one face) or float2 (two independent faces).
template <class V>
__device__ __forceinline__ void hllcv(const V L[5], const V R[5], const Gas& g, V F[5])
{
    const V pref = vbc<V>(g.pref), one = vbc<V>(1.0f);
    const V pL = vadd(L[1], pref), pR = vadd(R[1], pref);
    const V gpL = vmul(vbc<V>(g.gamma), pL), gpR = vmul(vbc<V>(g.gamma), pR);
    const V cL = vmul(gpL, vrsqrt(vmul(gpL, L[0])));
    const V cR = vmul(gpR, vrsqrt(vmul(gpR, R[0])));
    const V w = vmul(vmul(vsub(R[2], L[2]), vadd(L[0], R[0])), vadd(cL, cR));
    V pst = vfma(vbc<V>(-0.125f), w, vmul(vbc<V>(0.5f), vadd(L[1], R[1])));
    pst = vmaxs(pst, -g.pref);
    const V qL = vsqrt(vfma(vbc<V>(g.g1), vmaxs(vmul(vsub(pst, L[1]), vrcp(pL)), 0.0f), one));
    const V qR = vsqrt(vfma(vbc<V>(g.g1), vmaxs(vmul(vsub(pst, R[1]), vrcp(pR)), 0.0f), one));
    const V dsL = vneg(vmul(cL, qL));
    const V dsR = vmul(cR, qR);
    const V mL = vmul(L[0], dsL), mR = vmul(R[0], dsR);
    const V num = vsub(vfma(vneg(mR), R[2], R[1]), vfma(vneg(mL), L[2], L[1]));
    const V den = vsub(mL, mR);
    const auto left = vor(vge0(vadd(L[2], dsL)), vle0(num));  // s_L >= 0 or s_* >= 0
    const V rK = vsel(left, L[0], R[0]), pKd = vsel(left, L[1], R[1]), uK = vsel(left, L[2], R[2]);
    const V vK = vsel(left, L[3], R[3]), wK = vsel(left, L[4], R[4]);
    const V dsK = vsel(left, dsL, dsR), mK = vsel(left, mL, mR);
    const V pK = vadd(pKd, pref);
    const V sK = vadd(uK, dsK);
    const auto outer = vge0(vsel(left, sK, vneg(sK)));  // s_L >= 0, resp. s_R <= 0
    const V D = vfma(sK, den, vneg(num));
    const V r = vrcp(vmul(den, D));
    const V sst = vmul(num, vmul(D, r));
    const V inv = vmul(den, vmul(den, r));
    const V ke = vfma(wK, wK, vfma(vK, vK, vmul(uK, uK)));
    const V EK = vfma(pK, vbc<V>(g.igm1), vmul(vmul(vbc<V>(0.5f), rK), ke));
    const V phi = vmul(sst, inv);
    const V pstKd = vfma(mK, vsub(sst, uK), pKd);
    V F0 = vmul(phi, mK);
    V F1 = vfma(F0, sst, pstKd);
    const V A4 = vfma(EK, dsK, vneg(vmul(pK, uK)));
    V F4 = vmul(sst, vfma(A4, inv, vmul(vadd(pstKd, pref), vadd(one, phi))));
    const V G0 = vmul(rK, uK);
    const V G1 = vfma(G0, uK, pKd);
    const V G4 = vmul(vadd(EK, pK), uK);
    F0 = vsel(outer, G0, F0);
    F1 = vsel(outer, G1, F1);
    F4 = vsel(outer, G4, F4);
    F[0] = F0;
    F[1] = F1;
    F[2] = vmul(F0, vK);
    F[3] = vmul(F0, wK);
    F[4] = F4;
}

// Flux through faces whose normal is axis DIR, from states in the global frame (rho, p - pref, vx, vy, vz);
// result in conserved-field order (normal-momentum flux reduced by pref).
template <int DIR, class V>
__device__ __forceinline__ void face_fluxv(const V qL[5], const V qR[5], const Gas& g, V Fo[5])
{
    constexpr int iu = 2 + DIR, iv = 2 + (DIR + 1) % 3, iw = 2 + (DIR + 2) % 3;
    const V L[5] = {qL[0], qL[1], qL[iu], qL[iv], qL[iw]};
    const V R[5] = {qR[0], qR[1], qR[iu], qR[iv], qR[iw]};
    V F[5];
    hllcv<V>(L, R, g, F);
    Fo[0] = F[0];
    Fo[iu - 1] = F[1];
    Fo[iv - 1] = F[2];
    Fo[iw - 1] = F[3];
    Fo[4] = F[4];
}

template <int STAGE>
struct Smem {
    double2 raw[NRAW][5][PRP][PTX];                       // fp64 state of (row 2w, row 2w+1) at a column
    double2 u0[(STAGE == 2) ? 2 : 1][5][(STAGE == 2) ? PRP : 1][PTX];  // U0 of the planes being updated
    f2 Wt[2][5][PRP + 2][PTX + 4];                        // primitives, row pairs -1..PRP, columns -2..PTX+1
    f2 QLx[2][5][PRP][PTX + 1];                           // left states at x faces c = 0..PTX (from column c-1)
    float QLy[2][5][PRP + 1][PTX];                        // left states at the y faces between row pairs
    f2 Fx[2][5][PRP][PTX + 1];                            // float_t fluxes through x faces c = 0..PTX
    float Fy[2][5][PTY + 1][PTX];                         // float_t fluxes through y faces r = 0..PTY
    double red[32];
};

// One Heun stage of a 3D block.  STAGE 1: Uout = Uin + dt L(Uin).
// STAGE 2: Uout = 1/2 U0 + 1/2 (Uin + dt L(Uin)) (Uout may alias U0) and the CFL rate maximum of Uout.
template <int STAGE>
__global__ void __launch_bounds__(NTHREADS, 1)
stage_roles(const double* __restrict__ Uin, const double* U0, double* Uout, Grid g, Ctrl* ctrl, int zchunk)
{
    using S = Smem<STAGE>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    S& sm = *reinterpret_cast<S*>(smem_raw);

    const double dt = ctrl->dt;
    if (!(dt > 0.0)) return;  // a step clipped to zero length (run_until past t_end) does nothing
    const double pref_d = ctrl->p_ref;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int nx = g.n[0], ny = g.n[1], nz = g.n[2];
    const int i0 = blockIdx.x * PTX, j0 = blockIdx.y * PTY;
    const int kbeg = blockIdx.z * zchunk;
    const int kend = min(kbeg + zchunk, nz);
    const double gm1 = g.gamma - 1.0;
    const long long N = g.N;
    const long long pl = (long long)nx * ny;
    Gas gas;
    gas.gamma = (float)g.gamma;
    gas.g1 = (float)((g.gamma + 1.0) / (2.0 * g.gamma));
    gas.igm1 = (float)(1.0 / (g.gamma - 1.0));
    gas.pref = (float)pref_d;

    // strides (elements) of the shared arrays
    constexpr int RAWF = PRP * PTX, RAWS = 5 * RAWF;                       // double2: field, slot
    constexpr int WTR = PTX + 4, WTF = (PRP + 2) * WTR, WTB = 5 * WTF;     // f2: row, field, buffer
    constexpr int QXF = PRP * (PTX + 1), QXB = 5 * QXF;                    // f2 (QLx, Fx): field, buffer
    constexpr int QYF = (PRP + 1) * PTX, QYB = 5 * QYF;                    // float (QLy): field, buffer
    constexpr int FYF = (PTY + 1) * PTX, FYB = 5 * FYF;                    // float (Fy): field, buffer

    int hits = 0;
    f2 rate = pr::mk(0.0f, 0.0f);

    if (warp < WARP_XY0) {
        // ================================ ZU warps: columns (i, ja), (i, ja+1) ========================
        asm volatile("setmaxnreg.inc.sync.aligned.u32 " KH_ROLE_MAIN_REGS ";");
        const int w = warp;
        const int i = i0 + lane, ja = j0 + 2 * w;
        const bool in0 = (i < nx) && (ja < ny), in1 = (i < nx) && (ja + 1 < ny);
        int rx, rya, ryb;
        const int si = bc_source(i, nx, g.bc[0], g.bc[1], rx);
        const int sja = bc_source(ja, ny, g.bc[2], g.bc[3], rya);
        const int sjb = bc_source(ja + 1, ny, g.bc[2], g.bc[3], ryb);
        const int offa = sja * nx + si, offb = sjb * nx + si;  // < 2^31: checked at create
        const int cella = ja * nx + i;                         // valid when in0; the second cell is + nx

        double2* const raw0 = &sm.raw[0][0][w][lane];
        double2* const u00 = &sm.u0[0][0][(STAGE == 2) ? w : 0][lane];
        f2* const wt = &sm.Wt[0][0][w + 1][lane + 2];
        const f2* const fxs = &sm.Fx[0][0][w][lane];
        const float* const fys = &sm.Fy[0][0][2 * w][lane];

        const double dtdx = dt * g.inv_dx[0], dtdy = dt * g.inv_dx[1], dtdz = dt * g.inv_dx[2];
        const CflConst<float> cc(g);

        const int plo = kbeg - 2, phi = kend + 1;  // planes that exist for this slab
        auto fetch = [&](int kk, int slot) {
            if (kk < plo || kk > phi) return;
            int rz;
            const int sk = bc_source(kk, nz, g.bc[4], g.bc[5], rz);
            const double* a = Uin + (sk * pl + offa);
            const double* b = Uin + (sk * pl + offb);
            double2* d = raw0 + slot * RAWS;
#pragma unroll
            for (int f = 0; f < 5; f++) {
                pr::cp8(&d[f * RAWF].x, a + f * N);
                pr::cp8(&d[f * RAWF].y, b + f * N);
            }
        };
        auto fetch_u0 = [&](int kk) {
            if (STAGE != 2 || kk < kbeg || kk >= kend) return;
            const double* a = U0 + ((long long)kk * pl + cella);
            double2* d = u00 + (kk & 1) * RAWS;
#pragma unroll
            for (int f = 0; f < 5; f++) {
                if (in0) pr::cp8(&d[f * RAWF].x, a + f * N);
                if (in1) pr::cp8(&d[f * RAWF].y, a + nx + f * N);
            }
        };
        auto convert = [&](int kk, int slot, f2 W[5]) {
            int rz = VN_KEEP;
            (void)bc_source(kk, nz, g.bc[4], g.bc[5], rz);
            const double2* s = raw0 + slot * RAWS;
            double2 u[5];
#pragma unroll
            for (int f = 0; f < 5; f++) u[f] = s[f * RAWF];
            float Wa[5], Wb[5];
            const int ha = pr::recover(u[0].x, u[1].x, u[2].x, u[3].x, u[4].x, gm1, pref_d, rx, rya, rz, Wa);
            const int hb = pr::recover(u[0].y, u[1].y, u[2].y, u[3].y, u[4].y, gm1, pref_d, rx, ryb, rz, Wb);
            if (kk >= kbeg && kk < kend) hits += (in0 ? ha : 0) + (in1 ? hb : 0);
#pragma unroll
            for (int f = 0; f < 5; f++) W[f] = pr::mk(Wa[f], Wb[f]);
        };

        // ---- prologue: planes kbeg-2 .. kbeg in slots 0..2, plane kbeg+1 in slot 3 ----
        f2 Wa[5], Wb[5], QLz[5], Fzp[5];  // W(s), W(s+1), left state of z face s+1/2, flux through z face s-1/2
        fetch(kbeg - 2, 0);
        fetch(kbeg - 1, 1);
        fetch(kbeg, 2);
        __pipeline_commit();
        fetch(kbeg + 1, 3);
        __pipeline_commit();
        __pipeline_wait_prior(1);
        {
            f2 Wm[5];
            convert(kbeg - 2, 0, Wm);
            convert(kbeg - 1, 1, Wa);
            convert(kbeg, 2, Wb);
#pragma unroll
            for (int f = 0; f < 5; f++) {
                f2 qR;
                pr::plm(Wm[f], Wa[f], Wb[f], QLz[f], qR);
                Fzp[f] = pr::mk(0.0f, 0.0f);
            }
        }
        int s_new = 0;  // slot that receives plane s+3 (= slot of plane s-1)
        int s_conv = 3; // slot of plane s+2
        int s_upd = 1;  // slot of plane s

#pragma unroll 1
        for (int s = kbeg - 1; s < kend; s++) {
            // (1) publish the tile of plane s+1 for the XY and halo warps
            if (s + 1 < kend) {
                const int b = (s + 1) & 1;
                if (s - 1 >= kbeg) bar_sync(BAR_WT_FREE + b, CNT_ALL);  // plane s-1 has been read
                f2* const d = wt + b * WTB;
#pragma unroll
                for (int f = 0; f < 5; f++) d[f * WTF] = Wb[f];
                bar_arrive(BAR_WT_FULL + b, CNT_ALL);
            }
            // (2) next fetches; recover plane s+2; z face s+1/2
            fetch(s + 3, s_new);
            fetch_u0(s + 1);
            __pipeline_commit();
            __pipeline_wait_prior(1);  // plane s+2 (and U0 of plane s) have landed
            f2 Wn[5], Fzn[5];
            {
                convert(s + 2, s_conv, Wn);
                f2 qL[5], qR[5];
#pragma unroll
                for (int f = 0; f < 5; f++) {
                    qL[f] = QLz[f];
                    pr::plm(Wa[f], Wb[f], Wn[f], QLz[f], qR[f]);
                }
                face_fluxv<2, f2>(qL, qR, gas, Fzn);
            }
            // (3) fp64 update of plane s from the published x / y fluxes
            if (s >= kbeg) {
                const int b = s & 1;
                bar_sync(BAR_F_FULL + b, CNT_ALL);
                const double2* su = raw0 + s_upd * RAWS;
                const double2* s0 = u00 + b * RAWS;
                const f2* fx = fxs + b * QXB;
                const float* fy = fys + b * FYB;
                double* out = Uout + ((long long)s * pl + cella);
                double ua[5], ub[5];
#pragma unroll
                for (int f = 0; f < 5; f++) {
                    const f2 xl = fx[f * QXF], xh = fx[f * QXF + 1];
                    const float y0 = fy[f * FYF], y1 = fy[f * FYF + PTX], y2 = fy[f * FYF + 2 * PTX];
                    const double2 u = su[f * RAWF];
                    const double dy1 = (double)y1;
                    double da = dtdz * ((double)Fzp[f].x - (double)Fzn[f].x);
                    double db = dtdz * ((double)Fzp[f].y - (double)Fzn[f].y);
                    da = fma(dtdx, (double)xl.x - (double)xh.x, da);
                    db = fma(dtdx, (double)xl.y - (double)xh.y, db);
                    da = fma(dtdy, (double)y0 - dy1, da);
                    db = fma(dtdy, dy1 - (double)y2, db);
                    double xa = u.x + da, xb = u.y + db;
                    if (STAGE == 2) {
                        const double2 v = s0[f * RAWF];
                        xa = 0.5 * v.x + 0.5 * xa;
                        xb = 0.5 * v.y + 0.5 * xb;
                    }
                    ua[f] = xa;
                    ub[f] = xb;
                    if (in0) out[f * N] = xa;
                    if (in1) out[f * N + nx] = xb;
                }
                if (s + 2 < kend) bar_arrive(BAR_F_FREE + b, CNT_ALL);
                if (STAGE == 2) {
                    float ra = in0 ? cfl_rate_from_cons<float>(ua, cc) : 0.0f;
                    float rb = in1 ? cfl_rate_from_cons<float>(ub, cc) : 0.0f;
                    if (!(ra == ra)) ra = __int_as_float(0x7f800000);
                    if (!(rb == rb)) rb = __int_as_float(0x7f800000);
                    rate = pr::mk(fmaxf(rate.x, ra), fmaxf(rate.y, rb));
                }
            }
#pragma unroll
            for (int f = 0; f < 5; f++) { Wa[f] = Wb[f]; Wb[f] = Wn[f]; Fzp[f] = Fzn[f]; }
            s_new = (s_new == NRAW - 1) ? 0 : s_new + 1;
            s_conv = (s_conv == NRAW - 1) ? 0 : s_conv + 1;
            s_upd = (s_upd == NRAW - 1) ? 0 : s_upd + 1;
        }
        __pipeline_wait_prior(0);
    } else if (warp < WARP_H0) {
        // ================================ XY warps: x / y Riemann problems of the pair =================
        asm volatile("setmaxnreg.inc.sync.aligned.u32 " KH_ROLE_MAIN_REGS ";");
        const int w = warp - WARP_XY0;
        const f2* const wt = &sm.Wt[0][0][w + 1][lane + 2];
        f2* const qlx = &sm.QLx[0][0][w][lane];      // left state of the own low x face; own high face is + 1
        float* const qly = &sm.QLy[0][0][w][lane];   // left state of the pair's low y face; the pair's high face is + PTX
        f2* const fxs = &sm.Fx[0][0][w][lane];
        float* const fys = &sm.Fy[0][0][2 * w][lane];
#pragma unroll 1
        for (int k = kbeg; k < kend; k++) {
            const int b = k & 1;
            bar_sync(BAR_WT_FULL + b, CNT_ALL);
            // ---- phase A: x / y slopes of plane k (Eq. 3), left states published ----
            f2 QRx[5], QRy[5];
            float QLyo[5];  // left state of the face between the pair's two cells
            {
                const f2* const t = wt + b * WTB;
                f2* const qx = qlx + b * QXB;
                float* const qy = qly + b * QYB;
#pragma unroll
                for (int f = 0; f < 5; f++) {
                    const f2 q = t[f * WTF];
                    f2 qL;
                    pr::plm(t[f * WTF - 1], q, t[f * WTF + 1], qL, QRx[f]);
                    qx[f * QXF + 1] = qL;
                    const f2 below = t[f * WTF - WTR], above = t[f * WTF + WTR];
                    f2 qLy;
                    pr::plm(pr::mk(below.y, q.x), q, pr::mk(q.y, above.x), qLy, QRy[f]);
                    QLyo[f] = qLy.x;
                    qy[f * QYF + PTX] = qLy.y;
                }
            }
            if (k + 2 < kend) bar_arrive(BAR_WT_FREE + b, CNT_ALL);
            bar_sync(BAR_AB, CNT_AB);
            // ---- phase B: HLLC at the low x face and the two low y faces (Eq. 4-5) ----
            f2 Fxv[5], Fyv[5];
            {
                const f2* const qx = qlx + b * QXB;
                const float* const qy = qly + b * QYB;
                f2 qL[5];
#pragma unroll
                for (int f = 0; f < 5; f++) qL[f] = qx[f * QXF];
                face_fluxv<0, f2>(qL, QRx, gas, Fxv);
#pragma unroll
                for (int f = 0; f < 5; f++) qL[f] = pr::mk(qy[f * QYF], QLyo[f]);
                face_fluxv<1, f2>(qL, QRy, gas, Fyv);
            }
            if (k - 2 >= kbeg) bar_sync(BAR_F_FREE + b, CNT_ALL);  // the update of plane k-2 has read its fluxes
            {
                f2* const fx = fxs + b * QXB;
                float* const fy = fys + b * FYB;
#pragma unroll
                for (int f = 0; f < 5; f++) {
                    fx[f * QXF] = Fxv[f];
                    fy[f * FYF] = Fyv[f].x;
                    fy[f * FYF + PTX] = Fyv[f].y;
                }
            }
            bar_arrive(BAR_F_FULL + b, CNT_ALL);
        }
    } else {
        // ================================ halo warps ==================================================
        asm volatile("setmaxnreg.dec.sync.aligned.u32 " KH_ROLE_HALO_REGS ";");
        const int hw = warp - WARP_H0;  // 0: rows -2,-1   1: rows PTY,PTY+1   2: columns -2,-1   3: columns PTX,PTX+1
        if (hw < 2) {
            // ---- halo rows (lane = column): cells (c, r0), (c, r0+1) with r0 = -2 or PTY ----
            const int r0 = (hw == 0) ? -2 : PTY;
            int rx, ry0, ry1;
            const int si = bc_source(i0 + lane, nx, g.bc[0], g.bc[1], rx);
            const int sj0 = bc_source(j0 + r0, ny, g.bc[2], g.bc[3], ry0);
            const int sj1 = bc_source(j0 + r0 + 1, ny, g.bc[2], g.bc[3], ry1);
            const double* const src0 = Uin + ((long long)sj0 * nx + si);
            const double* const src1 = Uin + ((long long)sj1 * nx + si);
            f2* const wt = &sm.Wt[0][0][(hw == 0) ? 0 : PRP + 1][lane + 2];
            double u0v[5], u1v[5];
            auto load = [&](int kk) {
                const double* a = src0 + (long long)kk * pl;
                const double* c = src1 + (long long)kk * pl;
#pragma unroll
                for (int f = 0; f < 5; f++) { u0v[f] = __ldg(a + f * N); u1v[f] = __ldg(c + f * N); }
            };
            auto produce = [&](int kk) {  // tile rows of plane kk from the loaded state
                float W0[5], W1[5];
                (void)pr::recover(u0v[0], u0v[1], u0v[2], u0v[3], u0v[4], gm1, pref_d, rx, ry0, VN_KEEP, W0);
                (void)pr::recover(u1v[0], u1v[1], u1v[2], u1v[3], u1v[4], gm1, pref_d, rx, ry1, VN_KEEP, W1);
                const int b = kk & 1;
                if (kk - 2 >= kbeg) bar_sync(BAR_WT_FREE + b, CNT_ALL);
                f2* const d = wt + b * WTB;
#pragma unroll
                for (int f = 0; f < 5; f++) d[f * WTF] = pr::mk(W0[f], W1[f]);
            };
            load(kbeg);
            produce(kbeg);
            if (kbeg + 1 < kend) load(kbeg + 1);
#pragma unroll 1
            for (int k = kbeg; k < kend; k++) {
                const int b = k & 1;
                if (k + 1 < kend) {
                    produce(k + 1);
                    if (k + 2 < kend) load(k + 2);
                }
                bar_sync(BAR_WT_FULL + b, CNT_ALL);  // also announces this warp's rows of plane k
                // phase A: limited y state of the row next to the tile
                float qe[5];  // hw 1: right state of the tile's high y face
                {
                    const f2* const t = wt + b * WTB;
#pragma unroll
                    for (int f = 0; f < 5; f++) {
                        const f2 own = t[f * WTF];
                        float qL, qR;
                        if (hw == 0) {
                            const f2 r01 = t[f * WTF + WTR];        // rows 0, 1
                            vplm(own.x, own.y, r01.x, qL, qR);      // row -1
                            sm.QLy[b][f][0][lane] = qL;             // left state of the tile's low y face
                        } else {
                            const f2 rtop = t[f * WTF - WTR];       // rows PTY-2, PTY-1
                            vplm(rtop.y, own.x, own.y, qL, qR);     // row PTY
                            qe[f] = qR;
                        }
                    }
                }
                bar_sync(BAR_AB, CNT_AB);
                // phase B: flux through the tile's high y face
                float Fe[5];
                if (hw == 1) {
                    float qL[5];
#pragma unroll
                    for (int f = 0; f < 5; f++) qL[f] = sm.QLy[b][f][PRP][lane];
                    face_fluxv<1, float>(qL, qe, gas, Fe);
                }
                if (k - 2 >= kbeg) bar_sync(BAR_F_FREE + b, CNT_ALL);
                if (hw == 1) {
#pragma unroll
                    for (int f = 0; f < 5; f++) sm.Fy[b][f][PTY][lane] = Fe[f];
                }
                bar_arrive(BAR_F_FULL + b, CNT_ALL);
            }
        } else {
            // ---- halo columns: lane -> (row r = lane / 2, column c0 + lane % 2) with c0 = -2 or PTX ----
            const int cid = lane & 1, r = lane >> 1;
            const int col = ((hw == 2) ? -2 : PTX) + cid;
            int rx, ry;
            const int si = bc_source(i0 + col, nx, g.bc[0], g.bc[1], rx);
            const int sj = bc_source(j0 + r, ny, g.bc[2], g.bc[3], ry);
            const double* const src = Uin + ((long long)sj * nx + si);
            // element (row r, column col) of the f2 tile: pair r/2, component r%2
            float* const wt = reinterpret_cast<float*>(&sm.Wt[0][0][(r >> 1) + 1][col + 2]) + (r & 1);
            double uv[5];
            auto load = [&](int kk) {
                const double* a = src + (long long)kk * pl;
#pragma unroll
                for (int f = 0; f < 5; f++) uv[f] = __ldg(a + f * N);
            };
            auto produce = [&](int kk) {
                float W[5];
                (void)pr::recover(uv[0], uv[1], uv[2], uv[3], uv[4], gm1, pref_d, rx, ry, VN_KEEP, W);
                const int b = kk & 1;
                if (kk - 2 >= kbeg) bar_sync(BAR_WT_FREE + b, CNT_ALL);
                float* const d = wt + b * (2 * WTB);
#pragma unroll
                for (int f = 0; f < 5; f++) d[f * (2 * WTF)] = W[f];
            };
            const bool pub = (hw == 2) ? (cid == 1) : (cid == 0);  // the column next to the tile
            load(kbeg);
            produce(kbeg);
            if (kbeg + 1 < kend) load(kbeg + 1);
#pragma unroll 1
            for (int k = kbeg; k < kend; k++) {
                const int b = k & 1;
                if (k + 1 < kend) {
                    produce(k + 1);
                    if (k + 2 < kend) load(k + 2);
                }
                bar_sync(BAR_WT_FULL + b, CNT_ALL);
                // phase A: limited x state of the column next to the tile
                float qe[5];
                if (pub) {
                    const float* const t = wt + b * (2 * WTB);
#pragma unroll
                    for (int f = 0; f < 5; f++) {
                        float qL, qR;
                        vplm(t[f * (2 * WTF) - 2], t[f * (2 * WTF)], t[f * (2 * WTF) + 2], qL, qR);
                        if (hw == 2) reinterpret_cast<float*>(&sm.QLx[b][f][r >> 1][0])[r & 1] = qL;
                        else qe[f] = qR;
                    }
                }
                bar_sync(BAR_AB, CNT_AB);
                // phase B: flux through the tile's high x face
                float Fe[5];
                if (hw == 3 && pub) {
                    float qL[5];
#pragma unroll
                    for (int f = 0; f < 5; f++) qL[f] = reinterpret_cast<const float*>(&sm.QLx[b][f][r >> 1][PTX])[r & 1];
                    face_fluxv<0, float>(qL, qe, gas, Fe);
                }
                if (k - 2 >= kbeg) bar_sync(BAR_F_FREE + b, CNT_ALL);
                if (hw == 3 && pub) {
#pragma unroll
                    for (int f = 0; f < 5; f++) reinterpret_cast<float*>(&sm.Fx[b][f][r >> 1][PTX])[r & 1] = Fe[f];
                }
                bar_arrive(BAR_F_FULL + b, CNT_ALL);
            }
        }
    }

    if (hits) atomicAdd(&ctrl->floor_hits, (unsigned long long)hits);
    if (STAGE == 2) {
        __syncthreads();
        block_atomic_max_nonneg((double)fmaxf(rate.x, rate.y), &ctrl->rate_bits, sm.red);
    }
}

// ---------------------------------------------------------------------------------------
// host side
template <int STAGE>
inline void set_attr()
{
    static_assert(sizeof(Smem<STAGE>) <= 227 * 1024, "tile does not fit the shared memory of one SM");
    cudaFuncSetAttribute(stage_roles<STAGE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(Smem<STAGE>));
    cudaFuncSetAttribute(stage_roles<STAGE>, cudaFuncAttributePreferredSharedMemoryCarveout,
                         (int)cudaSharedmemCarveoutMaxShared);
}

inline void configure()
{
    set_attr<1>();
    set_attr<2>();
}

inline void launch_stage(int stage, const double* Uin, const double* U0, double* Uout, const Grid& g, Ctrl* ctrl,
                         int zchunk, cudaStream_t stream)
{
    dim3 grid((g.n[0] + PTX - 1) / PTX, (g.n[1] + PTY - 1) / PTY, (g.n[2] + zchunk - 1) / zchunk);
    if (stage == 1) stage_roles<1><<<grid, NTHREADS, sizeof(Smem<1>), stream>>>(Uin, U0, Uout, g, ctrl, zchunk);
    else            stage_roles<2><<<grid, NTHREADS, sizeof(Smem<2>), stream>>>(Uin, U0, Uout, g, ctrl, zchunk);
}

}  // namespace rl
}  // namespace kh
