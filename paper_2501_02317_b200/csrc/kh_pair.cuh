// kh_pair.cuh -- KRATOS_KERNEL_PAIRED: the fused Heun-stage kernel of the mixed-precision path
// (float_t = fp32, float2_t = fp64) for blocks with active x and y.
//
// The stage is limited by instruction issue, not by HBM, so this kernel is built
// to spend as few issue slots per cell as the scheme allows:
//   * every thread owns TWO cells, (i, 2w) and (i, 2w+1) of a 32 x 16 tile, and all float_t arithmetic
//     -- the minmod slopes of Eq. 3, the face states, the HLLC solver of Eq. 4-5 -- is done on the pair
//     with Blackwell's packed fp32 instructions (FADD2 / FMUL2 / FFMA2: two IEEE results per issue slot);
//     shared-memory traffic is 64 / 128 bit per access for the same reason;
//   * the 2-cell halo of the tile is loaded, converted, limited and (on the two high edges) solved by two
//     dedicated warps, so the eight main warps carry no halo code at all;
//   * every face flux is converted to float2_t once, by the thread that solved it, and handed to the
//     neighbouring cell in fp64;
//   * z is marched in registers (the column's primitives, its limited z state and the fp64 flux through
//     the last z face), the raw fp64 state of the thread's cells stays in a shared-memory ring from its
//     single fetch (cp.async, two planes ahead) to the fp64 update.
// Per plane: A) x/y slopes from the primitive tile, left states published | barrier | B) x/y/z fluxes,
// next plane's tile | barrier | C) fp64 update, Heun average and CFL rate of the new state (stage 2).
//
// Bit-identical fluxes across tile and slab seams: a face shared by two tiles (or slabs) is solved by both
// thread blocks.  Every operation on that path is explicitly rounded (no contraction, no re-association) and
// the special functions are single MUFU instructions, so both copies return the same bits and the fp64
// contributions to the two cells cancel exactly (conservation to float2_t accuracy).
#pragma once
#include <cuda_pipeline_primitives.h>

#include "kh_device.cuh"

namespace kh {
namespace pr {

typedef float2 f2;

constexpr int PTX = 32;            // tile width (one lane per column)
constexpr int PTY = 16;            // tile height
constexpr int PRP = PTY / 2;       // row pairs = main warps
constexpr int WARP_HALO_Y = PRP;       // rows -2,-1,PTY,PTY+1
constexpr int WARP_HALO_X = PRP + 1;   // columns -2,-1,PTX,PTX+1
constexpr int NWARPS = PRP + 4;        // two main warp groups + one halo warp group (its last two warps only keep the barriers)
constexpr int NTHREADS = NWARPS * 32;
// Register budget per scheduler: 2 main warps + 1 halo warp share 16384 registers (setmaxnreg below).
#define KH_PAIR_MAIN_REGS "184"
#define KH_PAIR_HALO_REGS "136"
constexpr int NSLOT = 5;           // raw ring depth: fetched at plane k-4, converted at k-2, updated at k

// ---- packed fp32 arithmetic, explicitly rounded --------------------------------------------------
__device__ __forceinline__ f2 mk(float a, float b) { return make_float2(a, b); }
__device__ __forceinline__ f2 bc(float s) { return make_float2(s, s); }
__device__ __forceinline__ f2 neg2(f2 a) { return make_float2(-a.x, -a.y); }
__device__ __forceinline__ f2 add2(f2 a, f2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ f2 sub2(f2 a, f2 b) { return __fadd2_rn(a, neg2(b)); }
__device__ __forceinline__ f2 mul2(f2 a, f2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ f2 fma2(f2 a, f2 b, f2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ f2 max0(f2 a) { return make_float2(fmaxf(a.x, 0.0f), fmaxf(a.y, 0.0f)); }
__device__ __forceinline__ f2 maxs(f2 a, float s) { return make_float2(fmaxf(a.x, s), fmaxf(a.y, s)); }
__device__ __forceinline__ f2 rcp2(f2 a) { return make_float2(rcp_(a.x), rcp_(a.y)); }
__device__ __forceinline__ f2 sqrt2(f2 a) { return make_float2(sqrt_(a.x), sqrt_(a.y)); }
__device__ __forceinline__ f2 rsqrt2(f2 a) { return make_float2(rsqrt_(a.x), rsqrt_(a.y)); }
__device__ __forceinline__ f2 sel(bool cx, bool cy, f2 a, f2 b) { return make_float2(cx ? a.x : b.x, cy ? a.y : b.y); }
__device__ __forceinline__ f2 mm2(f2 a, f2 b) { return make_float2(minmod(a.x, b.x), minmod(a.y, b.y)); }

// Face states of a cell from its value q and its two undivided differences a = q - q_minus, b = q_plus - q
// (Eq. 3; reading S8): qL = q + minmod(a,b)/2 (left state of the high face),
// qR = q - minmod(a,b)/2 (right state of the low face).  The product with 1/2 is exact, so the fused form
// rounds once, exactly like q +- h.
__device__ __forceinline__ void plm(f2 qm, f2 q, f2 qp, f2& qL, f2& qR)
{
    const f2 s = mm2(sub2(q, qm), sub2(qp, q));
    qL = fma2(bc(0.5f), s, q);
    qR = fma2(bc(-0.5f), s, q);
}

// The same for a pair of cells that are neighbours along the axis (rows 2w, 2w+1 of a column): face states of both from the
// four values below, q.x, q.y, above.  Operation for operation plm(mk(below, q.x), q, mk(q.y, above), ...): the three undivided
// differences are formed once, as scalars (the packed form has to assemble two shifted register pairs first: four moves).
__device__ __forceinline__ void plm_along_pair(float below, f2 q, float above, f2& qL, f2& qR)
{
    const float d0 = __fadd_rn(q.x, -below), d1 = __fadd_rn(q.y, -q.x), d2 = __fadd_rn(above, -q.y);
    const f2 s = mk(minmod(d0, d1), minmod(d1, d2));
    qL = fma2(bc(0.5f), s, q);
    qR = fma2(bc(-0.5f), s, q);
}

struct Gas {
    float gamma, g1, igm1, pref;
};

// Sec. 3.2.2: HLLC with the wave speeds of Eq. 5 and the contact speed of Eq. 4, for
// two independent faces at once.  Same formulas, same order of operations as kh::hllc (kh_device.cuh),
// where they are documented; states are (rho, p - pref, u, v, w) with u normal to the face, the result is
// (mass, normal momentum - pref, tangential 1, tangential 2, energy).
__device__ __forceinline__ void hllc2(const f2 L[5], const f2 R[5], const Gas& g, f2 F[5])
{
    const f2 pref = bc(g.pref);
    const f2 pL = add2(L[1], pref), pR = add2(R[1], pref);
    const f2 gpL = mul2(bc(g.gamma), pL), gpR = mul2(bc(g.gamma), pR);
    const f2 tL = rsqrt2(mul2(gpL, L[0])), tR = rsqrt2(mul2(gpR, R[0]));
    const f2 cL = mul2(gpL, tL), cR = mul2(gpR, tR);
    const f2 w = mul2(mul2(sub2(R[2], L[2]), add2(L[0], R[0])), add2(cL, cR));
    f2 pst = fma2(bc(-0.125f), w, mul2(bc(0.5f), add2(L[1], R[1])));
    pst = maxs(pst, -g.pref);
    const f2 one = bc(1.0f);
    // 1/p_K = gamma rho_K t_K^2 with t_K = rsqrt(gamma p_K rho_K) from the sound speed (see tma::hllc2n)
    const f2 ipL = mul2(mul2(bc(g.gamma), L[0]), mul2(tL, tL)), ipR = mul2(mul2(bc(g.gamma), R[0]), mul2(tR, tR));
    const f2 qL = sqrt2(fma2(bc(g.g1), max0(mul2(sub2(pst, L[1]), ipL)), one));
    const f2 qR = sqrt2(fma2(bc(g.g1), max0(mul2(sub2(pst, R[1]), ipR)), one));
    const f2 dsL = neg2(mul2(cL, qL));
    const f2 dsR = mul2(cR, qR);
    const f2 mL = mul2(L[0], dsL), mR = mul2(R[0], dsR);
    const f2 num = sub2(fma2(neg2(mR), R[2], R[1]), fma2(neg2(mL), L[2], L[1]));
    const f2 den = sub2(mL, mR);
    const f2 sL = add2(L[2], dsL);
    const bool lx = (sL.x >= 0.0f) || (num.x <= 0.0f), ly = (sL.y >= 0.0f) || (num.y <= 0.0f);
    const f2 rK = sel(lx, ly, L[0], R[0]), pKd = sel(lx, ly, L[1], R[1]), uK = sel(lx, ly, L[2], R[2]);
    const f2 vK = sel(lx, ly, L[3], R[3]), wK = sel(lx, ly, L[4], R[4]);
    const f2 dsK = sel(lx, ly, dsL, dsR), mK = sel(lx, ly, mL, mR);
    const f2 pK = add2(pKd, pref);
    const f2 sK = add2(uK, dsK);
    const bool ox = (lx ? sK.x : -sK.x) >= 0.0f, oy = (ly ? sK.y : -sK.y) >= 0.0f;
    const f2 D = fma2(sK, den, neg2(num));
    const f2 r = rcp2(mul2(den, D));
    const f2 sst = mul2(num, mul2(D, r));
    const f2 inv = mul2(den, mul2(den, r));
    const f2 ke = fma2(wK, wK, fma2(vK, vK, mul2(uK, uK)));
    const f2 EK = fma2(pK, bc(g.igm1), mul2(mul2(bc(0.5f), rK), ke));
    const f2 phi = mul2(sst, inv);
    const f2 pstKd = fma2(mK, sub2(sst, uK), pKd);
    f2 F0 = mul2(phi, mK);
    f2 F1 = fma2(F0, sst, pstKd);
    const f2 A4 = fma2(EK, dsK, neg2(mul2(pK, uK)));
    f2 F4 = mul2(sst, fma2(A4, inv, mul2(add2(pstKd, pref), add2(one, phi))));
    const f2 G0 = mul2(rK, uK);
    const f2 G1 = fma2(G0, uK, pKd);
    const f2 G4 = mul2(add2(EK, pK), uK);
    F0 = sel(ox, oy, G0, F0);
    F1 = sel(ox, oy, G1, F1);
    F4 = sel(ox, oy, G4, F4);
    F[0] = F0;
    F[1] = F1;
    F[2] = mul2(F0, vK);
    F[3] = mul2(F0, wK);
    F[4] = F4;
}

// Flux through two faces whose normal is axis DIR, from states in the global frame
// (rho, p - pref, vx, vy, vz); result in conserved-field order (normal-momentum flux reduced by pref).
template <int DIR>
__device__ __forceinline__ void face_flux2(const f2 qL[5], const f2 qR[5], const Gas& g, f2 Fo[5])
{
    constexpr int iu = 2 + DIR, iv = 2 + (DIR + 1) % 3, iw = 2 + (DIR + 2) % 3;
    const f2 L[5] = {qL[0], qL[1], qL[iu], qL[iv], qL[iw]};
    const f2 R[5] = {qR[0], qR[1], qR[iu], qR[iv], qR[iw]};
    f2 F[5];
    hllc2(L, R, g, F);
    Fo[0] = F[0];
    Fo[iu - 1] = F[1];
    Fo[iv - 1] = F[2];
    Fo[iw - 1] = F[3];
    Fo[4] = F[4];
}

// Sec. 3.1, reading S7: fp64 recovery of (rho, p - pref, v) of one cell, explicitly
// rounded so that every copy (main warps, halo warps, neighbouring blocks) returns the same bits;
// 1/rho by MUFU.RCP64H + one Newton step (2^-40, far below the fp32 rounding of the result).
// Boundary rules act on the normal velocities.  Returns the floor activations (S6).
// With a reference pressure the floor is max(1e-30, pref 2^-22): two fp32 ulps of pref, so that the stored
// deviation p - pref never rounds to -pref and the pressure rebuilt by the Riemann solver stays > 0 (the
// limited face states lie between the cell values, Eq. 3).  pref <= 2 p_min when it is set (kh_reduce.cuh),
// so this floor is 5e-7 of the lowest pressure the block held then.
__device__ __forceinline__ int recover(double rho, double mx, double my, double mz, double e, double gm1, double pref,
                                       int rx, int ry, int rz, float W[5])
{
    const bool lo_r = rho < KH_RHO_FLOOR;
    rho = lo_r ? KH_RHO_FLOOR : rho;
    double ir;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(ir) : "d"(rho));
    ir = __fma_rn(ir, __fma_rn(-rho, ir, 1.0), ir);
    double vx = __dmul_rn(mx, ir), vy = __dmul_rn(my, ir), vz = __dmul_rn(mz, ir);
    // (m.m)/rho with m.m formed first: it does not wait for the reciprocal, which shortens the dependent chain
    const double m2 = __dmul_rn(__fma_rn(mz, mz, __fma_rn(my, my, __dmul_rn(mx, mx))), ir);
    double p = __dmul_rn(gm1, __fma_rn(-0.5, m2, e));
    const double pfl = fmax(KH_P_FLOOR, __dmul_rn(pref, 0x1p-22));
    const bool lo_p = p < pfl;
    p = lo_p ? pfl : p;
    if (rx | ry | rz) {
        vx = apply_vn_rule(vx, rx);
        vy = apply_vn_rule(vy, ry);
        vz = apply_vn_rule(vz, rz);
    }
    W[0] = (float)rho;
    W[1] = (float)__dadd_rn(p, -pref);
    W[2] = (float)vx;
    W[3] = (float)vy;
    W[4] = (float)vz;
    return (int)lo_r + (int)lo_p;
}

// All-fp32 "Single" mode (float2_t = float_t = float): the recovery on an fp32 state, in fp32
// (kh::cons_to_prim(float...): explicitly rounded, 1/rho by MUFU.RCP); no reference pressure (pref = 0).
__device__ __forceinline__ int recover(float rho, float mx, float my, float mz, float e, float gm1, float pref, int rx, int ry,
                                       int rz, float W[5])
{
    float p, vx, vy, vz, r;
    const int hits = cons_to_prim(rho, mx, my, mz, e, gm1, p, vx, vy, vz, r);
    W[0] = r;
    W[1] = __fadd_rn(p, -pref);
    W[2] = apply_vn_rule(vx, rx);
    W[3] = apply_vn_rule(vy, ry);
    W[4] = apply_vn_rule(vz, rz);
    return hits;
}

template <int STAGE>
struct Smem {
    double2 raw[NSLOT][5][PRP][PTX];                          // fp64 state of (row 2w, row 2w+1) at a column
    double2 u0[(STAGE == 2) ? 2 : 1][5][(STAGE == 2) ? PRP : 1][PTX];  // U0 of the plane being updated
    f2 Wt[5][PRP + 2][PTX + 4];                               // primitives of one plane, row pairs -1..PRP, columns -2..PTX+1
    f2 QLx[5][PRP][PTX + 1];                                  // left states at x faces c = 0..PTX (from column c-1)
    f2 QRxR[5][PRP];                                          // right state at x face PTX (from halo column PTX)
    float QLy[5][PRP + 1][PTX];                               // left states at y faces r = 0..PRP (from row 2r-1)
    float QRyT[5][PTX];                                       // right state at y face PRP (from halo row PTY)
    double2 Fx[5][PRP][PTX + 1];                              // fp64 fluxes through x faces
    double Fy[5][PRP + 1][PTX];                               // fp64 fluxes through the y faces between row pairs
    double red[32];
};

__device__ __forceinline__ void block_bar() { asm volatile("bar.sync 0;" ::: "memory"); }

__device__ __forceinline__ void cp8(void* smem_dst, const void* gmem_src) { __pipeline_memcpy_async(smem_dst, gmem_src, 8); }

// One Heun stage.  STAGE 1: Uout = Uin + dt L(Uin).  STAGE 2: Uout = 1/2 U0 + 1/2 (Uin + dt L(Uin))
// (Uout may alias U0) and the CFL rate maximum of Uout.  NDIM = 2 (nz == 1) or 3.
template <int STAGE, int NDIM>
__global__ void __launch_bounds__(NTHREADS, 1)
stage_pair(const double* __restrict__ Uin, const double* U0, double* Uout, Grid g, Ctrl* ctrl, int zchunk)
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
    const int kbeg = (NDIM == 3) ? blockIdx.z * zchunk : 0;
    const int kend = (NDIM == 3) ? min(kbeg + zchunk, nz) : 1;
    const int kfirst = (NDIM == 3) ? kbeg - 1 : -1;  // priming iteration: builds the tile of plane kbeg
    const double gm1 = g.gamma - 1.0;
    const long long N = g.N;
    const long long pl = (long long)nx * ny;
    Gas gas;
    gas.gamma = (float)g.gamma;
    gas.g1 = (float)((g.gamma + 1.0) / (2.0 * g.gamma));
    gas.igm1 = (float)(1.0 / (g.gamma - 1.0));
    gas.pref = (float)pref_d;

    int hits = 0;
    f2 rate = mk(0.0f, 0.0f);

    if (warp < PRP) {
        // ================================ main warps: cells (i, ja), (i, ja+1) ========================
        asm volatile("setmaxnreg.inc.sync.aligned.u32 " KH_PAIR_MAIN_REGS ";");
        const int w = warp;
        const int i = i0 + lane, ja = j0 + 2 * w;
        const bool in0 = (i < nx) && (ja < ny), in1 = (i < nx) && (ja + 1 < ny);
        int rx, rya, ryb;
        const int si = bc_source(i, nx, g.bc[0], g.bc[1], rx);
        const int sja = bc_source(ja, ny, g.bc[2], g.bc[3], rya);
        const int sjb = bc_source(ja + 1, ny, g.bc[2], g.bc[3], ryb);
        // element offsets inside one plane of one field (< 2^31: checked at create)
        const int offa = sja * nx + si, offb = sjb * nx + si;
        const int cella = ja * nx + i;  // valid when in0; the pair's second cell is + nx

        constexpr int RAWF = PRP * PTX, RAWS = 5 * RAWF;              // double2 strides of raw / u0: field, slot
        constexpr int WTF = (PRP + 2) * (PTX + 4);                    // f2 field stride of Wt
        constexpr int QXF = PRP * (PTX + 1);                          // f2 field stride of QLx, double2 of Fx
        constexpr int QYF = (PRP + 1) * PTX;                          // field stride of QLy (float) and Fy (double)
        double2* const raw0 = &sm.raw[0][0][w][lane];
        double2* const u00 = &sm.u0[0][0][(STAGE == 2) ? w : 0][lane];
        f2* const wt = &sm.Wt[0][w + 1][lane + 2];
        f2* const qlx = &sm.QLx[0][w][lane];      // left state of the own low x face; own high face is + 1
        float* const qly = &sm.QLy[0][w][lane];   // left state of the pair's low y face; the pair's high face is + PTX
        double2* const fxs = &sm.Fx[0][w][lane];
        double* const fys = &sm.Fy[0][w][lane];

        const double dtdx = dt * g.inv_dx[0], dtdy = dt * g.inv_dx[1], dtdz = dt * g.inv_dx[2];
        const CflConst<float> cc(g);

        // planes that exist for this slab: the slab itself plus two stencil planes on either side
        const int plo = (NDIM == 3) ? kbeg - 2 : 0, phi = (NDIM == 3) ? kend + 1 : 0;
        auto fetch = [&](int kk, int slot) {
            if (kk < plo || kk > phi) return;
            int rz;
            const int sk = (NDIM == 3) ? bc_source(kk, nz, g.bc[4], g.bc[5], rz) : 0;
            const double* a = Uin + (sk * pl + offa);
            const double* b = Uin + (sk * pl + offb);
            double2* d = raw0 + slot * RAWS;
#pragma unroll
            for (int f = 0; f < 5; f++) {
                cp8(&d[f * RAWF].x, a + f * N);
                cp8(&d[f * RAWF].y, b + f * N);
            }
        };
        auto fetch_u0 = [&](int kk) {
            if (STAGE != 2 || kk < kbeg || kk >= kend) return;
            const double* a = U0 + ((long long)kk * pl + cella);
            double2* d = u00 + (kk & 1) * RAWS;
#pragma unroll
            for (int f = 0; f < 5; f++) {
                if (in0) cp8(&d[f * RAWF].x, a + f * N);
                if (in1) cp8(&d[f * RAWF].y, a + nx + f * N);
            }
        };
        auto convert = [&](int kk, int slot, f2 W[5]) {
            int rz = VN_KEEP;
            if (NDIM == 3) (void)bc_source(kk, nz, g.bc[4], g.bc[5], rz);
            const double2* s = raw0 + slot * RAWS;
            double2 u[5];
#pragma unroll
            for (int f = 0; f < 5; f++) u[f] = s[f * RAWF];
            float Wa[5], Wb[5];
            const int ha = recover(u[0].x, u[1].x, u[2].x, u[3].x, u[4].x, gm1, pref_d, rx, rya, rz, Wa);
            const int hb = recover(u[0].y, u[1].y, u[2].y, u[3].y, u[4].y, gm1, pref_d, rx, ryb, rz, Wb);
            if (kk >= kbeg && kk < kend) hits += (in0 ? ha : 0) + (in1 ? hb : 0);
#pragma unroll
            for (int f = 0; f < 5; f++) W[f] = mk(Wa[f], Wb[f]);
        };

        // ---- prologue ----
        f2 Wa[5], Wb[5], QLz[5];   // W(k), W(k+1), left state of z face k+1/2
        double2 Fzlo[5];           // dt/dz * flux through z face k-1/2
        int s_fetch, s_conv, s_upd;  // ring slots of the planes k+4, k+2, k
        if (NDIM == 3) {
            fetch(kbeg - 2, 0);
            fetch(kbeg - 1, 1);
            fetch(kbeg, 2);
            __pipeline_commit();
            fetch(kbeg + 1, 3);
            __pipeline_commit();
            fetch(kbeg + 2, 4);
            __pipeline_commit();
            __pipeline_wait_prior(2);
            f2 Wm[5];
            convert(kbeg - 2, 0, Wm);
            convert(kbeg - 1, 1, Wa);
            convert(kbeg, 2, Wb);
#pragma unroll
            for (int f = 0; f < 5; f++) {
                f2 qR;
                plm(Wm[f], Wa[f], Wb[f], QLz[f], qR);
                Fzlo[f] = make_double2(0.0, 0.0);
            }
            s_fetch = 0;  // plane kfirst+4 = kbeg+3 reuses the slot of plane kbeg-2
            s_conv = 3;   // plane kfirst+2 = kbeg+1
            s_upd = 1;    // plane kfirst = kbeg-1 (never updated)
        } else {
            fetch(0, 0);
            __pipeline_commit();
            __pipeline_commit();
            __pipeline_commit();
            __pipeline_wait_prior(2);
            convert(0, 0, Wb);
#pragma unroll
            for (int f = 0; f < 5; f++) {
                Wa[f] = Wb[f];
                QLz[f] = Wb[f];
                Fzlo[f] = make_double2(0.0, 0.0);
            }
            s_fetch = 1;
            s_conv = 1;
            s_upd = 4;  // becomes 0 for plane 0
        }

        f2 QRx[5], QRy[5];
        float QLyo[5];  // left state of the face between the pair's two cells
        double2 dU[5];
#pragma unroll
        for (int f = 0; f < 5; f++) { QRx[f] = QRy[f] = mk(0.f, 0.f); QLyo[f] = 0.f; dU[f] = make_double2(0.0, 0.0); }

#pragma unroll 1
        for (int k = kfirst; k < kend; k++) {
            const bool live = k >= kbeg;
            // ---------------- phase A: x / y slopes of plane k from the tile ----------------
            if (live) {
#pragma unroll
                for (int f = 0; f < 5; f++) {
                    const f2 q = Wa[f];
                    f2 qL;
                    plm(wt[f * WTF - 1], q, wt[f * WTF + 1], qL, QRx[f]);
                    qlx[f * QXF + 1] = qL;
                    const f2 below = wt[f * WTF - (PTX + 4)], above = wt[f * WTF + (PTX + 4)];
                    f2 qLy;
                    plm_along_pair(below.y, q, above.x, qLy, QRy[f]);
                    QLyo[f] = qLy.x;
                    qly[f * QYF + PTX] = qLy.y;
                }
            }
            block_bar();
            // ---------------- phase B: fluxes of plane k, tile of plane k+1 ----------------
            fetch(k + 4, s_fetch);
            fetch_u0(k + 1);
            __pipeline_commit();
            f2 Wn[5];
            double2 Fzhi[5];
            if (NDIM == 3) {
                __pipeline_wait_prior(2);
                convert(k + 2, s_conv, Wn);
                f2 qL[5], qR[5], F[5];
#pragma unroll
                for (int f = 0; f < 5; f++) {
                    qL[f] = QLz[f];
                    plm(Wa[f], Wb[f], Wn[f], QLz[f], qR[f]);
                }
                face_flux2<2>(qL, qR, gas, F);
#pragma unroll
                for (int f = 0; f < 5; f++) {
                    Fzhi[f] = make_double2(dtdz * (double)F[f].x, dtdz * (double)F[f].y);
                    dU[f] = make_double2(Fzlo[f].x - Fzhi[f].x, Fzlo[f].y - Fzhi[f].y);
                }
            }
            if (live) {
                {
                    f2 qL[5], F[5];
#pragma unroll
                    for (int f = 0; f < 5; f++) qL[f] = qlx[f * QXF];
                    face_flux2<0>(qL, QRx, gas, F);
#pragma unroll
                    for (int f = 0; f < 5; f++) {
                        const double2 fd = make_double2((double)F[f].x, (double)F[f].y);
                        fxs[f * QXF] = fd;
                        dU[f].x = fma(dtdx, fd.x, dU[f].x);
                        dU[f].y = fma(dtdx, fd.y, dU[f].y);
                    }
                }
                {
                    f2 qL[5], F[5];
#pragma unroll
                    for (int f = 0; f < 5; f++) qL[f] = mk(qly[f * QYF], QLyo[f]);
                    face_flux2<1>(qL, QRy, gas, F);
#pragma unroll
                    for (int f = 0; f < 5; f++) {
                        const double flo = (double)F[f].x, fin = (double)F[f].y;
                        fys[f * QYF] = flo;
                        dU[f].x = fma(dtdy, flo - fin, dU[f].x);
                        dU[f].y = fma(dtdy, fin, dU[f].y);
                    }
                }
            }
            if (k + 1 < kend) {
#pragma unroll
                for (int f = 0; f < 5; f++) wt[f * WTF] = Wb[f];
            }
            block_bar();
            // ---------------- phase C: fp64 update of plane k ----------------
            if (live) {
                if (STAGE == 2) __pipeline_wait_prior(1);  // U0(k) has landed (this thread's own copies)
                const double2* su = raw0 + s_upd * RAWS;
                const double2* s0 = u00 + (k & 1) * RAWS;
                double* out = Uout + ((long long)k * pl + cella);
                double ua[5], ub[5];
#pragma unroll
                for (int f = 0; f < 5; f++) {
                    const double2 fxh = fxs[f * QXF + 1];
                    const double fyh = fys[f * QYF + PTX];
                    const double2 u = su[f * RAWF];
                    double xa = u.x + fma(-dtdx, fxh.x, dU[f].x);
                    double xb = u.y + fma(-dtdy, fyh, fma(-dtdx, fxh.y, dU[f].y));
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
                if (STAGE == 2) {
                    float ra = in0 ? cfl_rate_from_cons<float>(ua, cc) : 0.0f;
                    float rb = in1 ? cfl_rate_from_cons<float>(ub, cc) : 0.0f;
                    if (!(ra == ra)) ra = __int_as_float(0x7f800000);
                    if (!(rb == rb)) rb = __int_as_float(0x7f800000);
                    rate = mk(fmaxf(rate.x, ra), fmaxf(rate.y, rb));
                }
            }
            // rotate the z march and the ring
#pragma unroll
            for (int f = 0; f < 5; f++) {
                Wa[f] = Wb[f];
                if (NDIM == 3) { Wb[f] = Wn[f]; Fzlo[f] = Fzhi[f]; }
            }
            s_fetch = (s_fetch == NSLOT - 1) ? 0 : s_fetch + 1;
            s_conv = (s_conv == NSLOT - 1) ? 0 : s_conv + 1;
            s_upd = (s_upd == NSLOT - 1) ? 0 : s_upd + 1;
        }
        __pipeline_wait_prior(0);
    } else {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 " KH_PAIR_HALO_REGS ";");
        if (warp == WARP_HALO_Y) {
        // ================================ halo rows -2, -1, PTY, PTY+1 (lane = column) ==================
        const int i = i0 + lane;
        int rx, ry[4];
        const int si = bc_source(i, nx, g.bc[0], g.bc[1], rx);
        const double* src[4];
#pragma unroll
        for (int r = 0; r < 4; r++) {
            const int row = (r < 2) ? r - 2 : PTY + r - 2;
            const int sj = bc_source(j0 + row, ny, g.bc[2], g.bc[3], ry[r]);
            src[r] = Uin + ((long long)sj * nx + si);
        }
        constexpr int WTF = (PRP + 2) * (PTX + 4);
        constexpr int QYF = (PRP + 1) * PTX;
        f2* const wlo = &sm.Wt[0][0][lane + 2];          // rows -2, -1
        f2* const whi = &sm.Wt[0][PRP + 1][lane + 2];    // rows PTY, PTY+1
        double u[4][5];
        auto load = [&](int kk) {
            const double* base = nullptr;
#pragma unroll
            for (int r = 0; r < 4; r++) {
                base = src[r] + (long long)kk * pl;
#pragma unroll
                for (int f = 0; f < 5; f++) u[r][f] = __ldg(base + f * N);
            }
        };
        float W[4][5];
#pragma unroll
        for (int r = 0; r < 4; r++)
#pragma unroll
            for (int f = 0; f < 5; f++) W[r][f] = 0.0f;
        load(kbeg);
#pragma unroll 1
        for (int k = kfirst; k < kend; k++) {
            const bool live = k >= kbeg;
            // phase A: limited y states of rows -1 and PTY of plane k
            if (live) {
#pragma unroll
                for (int f = 0; f < 5; f++) {
                    const f2 r01 = wlo[f * WTF + (PTX + 4)];        // rows 0, 1
                    const f2 rtop = whi[f * WTF - (PTX + 4)];       // rows PTY-2, PTY-1
                    f2 qL, qR;
                    plm(mk(W[0][f], rtop.y), mk(W[1][f], W[2][f]), mk(r01.x, W[3][f]), qL, qR);
                    sm.QLy[f][0][lane] = qL.x;    // row -1: left state of the tile's low y face
                    sm.QRyT[f][lane] = qR.y;      // row PTY: right state of the tile's high y face
                }
            }
            block_bar();
            // phase B: flux through the tile's high y face of plane k; halo rows of plane k+1
            if (live) {
                f2 qL[5], qR[5], F[5];
#pragma unroll
                for (int f = 0; f < 5; f++) {
                    const float l = sm.QLy[f][PRP][lane], r = sm.QRyT[f][lane];
                    qL[f] = mk(l, l);
                    qR[f] = mk(r, r);
                }
                face_flux2<1>(qL, qR, gas, F);
#pragma unroll
                for (int f = 0; f < 5; f++) sm.Fy[f][PRP][lane] = (double)F[f].x;
            }
            if (k + 1 < kend) {
#pragma unroll
                for (int r = 0; r < 4; r++)
                    (void)recover(u[r][0], u[r][1], u[r][2], u[r][3], u[r][4], gm1, pref_d, rx, ry[r], VN_KEEP, W[r]);
#pragma unroll
                for (int f = 0; f < 5; f++) {
                    wlo[f * WTF] = mk(W[0][f], W[1][f]);
                    whi[f * WTF] = mk(W[2][f], W[3][f]);
                }
                if (k + 2 < kend) load(k + 2);
            }
            block_bar();
        }
    } else if (warp == WARP_HALO_X) {
        // ================================ halo columns -2, -1, PTX, PTX+1 =============================
        const int cid = lane & 3, rp = lane >> 2;                   // column id, row pair
        const int col = (cid < 2) ? cid - 2 : PTX + cid - 2;
        const int ja = j0 + 2 * rp;
        int rx, rya, ryb;
        const int si = bc_source(i0 + col, nx, g.bc[0], g.bc[1], rx);
        const int sja = bc_source(ja, ny, g.bc[2], g.bc[3], rya);
        const int sjb = bc_source(ja + 1, ny, g.bc[2], g.bc[3], ryb);
        const double* const srca = Uin + ((long long)sja * nx + si);
        const double* const srcb = Uin + ((long long)sjb * nx + si);
        constexpr int WTF = (PRP + 2) * (PTX + 4);
        f2* const wt = &sm.Wt[0][rp + 1][col + 2];
        const int dl = (cid == 0) ? 0 : -1, dr = (cid == 3) ? 0 : 1;   // neighbours inside the tile array
        double ua[5], ub[5];
        auto load = [&](int kk) {
            const double* a = srca + (long long)kk * pl;
            const double* b = srcb + (long long)kk * pl;
#pragma unroll
            for (int f = 0; f < 5; f++) { ua[f] = __ldg(a + f * N); ub[f] = __ldg(b + f * N); }
        };
        f2 W[5];
#pragma unroll
        for (int f = 0; f < 5; f++) W[f] = mk(0.f, 0.f);
        load(kbeg);
#pragma unroll 1
        for (int k = kfirst; k < kend; k++) {
            const bool live = k >= kbeg;
            // phase A: limited x states of columns -1 and PTX of plane k
            if (live) {
#pragma unroll
                for (int f = 0; f < 5; f++) {
                    f2 qL, qR;
                    plm(wt[f * WTF + dl], W[f], wt[f * WTF + dr], qL, qR);
                    if (cid == 1) sm.QLx[f][rp][0] = qL;   // column -1: left state of the tile's low x face
                    if (cid == 2) sm.QRxR[f][rp] = qR;     // column PTX: right state of the tile's high x face
                }
            }
            block_bar();
            // phase B: flux through the tile's high x face of plane k; halo columns of plane k+1
            if (live && cid == 2) {
                f2 qL[5], qR[5], F[5];
#pragma unroll
                for (int f = 0; f < 5; f++) { qL[f] = sm.QLx[f][rp][PTX]; qR[f] = sm.QRxR[f][rp]; }
                face_flux2<0>(qL, qR, gas, F);
#pragma unroll
                for (int f = 0; f < 5; f++) sm.Fx[f][rp][PTX] = make_double2((double)F[f].x, (double)F[f].y);
            }
            if (k + 1 < kend) {
                float Wa[5], Wb[5];
                (void)recover(ua[0], ua[1], ua[2], ua[3], ua[4], gm1, pref_d, rx, rya, VN_KEEP, Wa);
                (void)recover(ub[0], ub[1], ub[2], ub[3], ub[4], gm1, pref_d, rx, ryb, VN_KEEP, Wb);
#pragma unroll
                for (int f = 0; f < 5; f++) {
                    W[f] = mk(Wa[f], Wb[f]);
                    wt[f * WTF] = W[f];
                }
                if (k + 2 < kend) load(k + 2);
            }
            block_bar();
        }
    } else {
#pragma unroll 1
        for (int k = kfirst; k < kend; k++) { block_bar(); block_bar(); }
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
inline int auto_zchunk(const Grid& g)
{
    if (!g.active[2]) return 1;
    // >= ~12 waves of thread blocks over the SMs (148 on B200; one block per SM), slabs of >= 32 planes
    const long long tiles = (long long)((g.n[0] + PTX - 1) / PTX) * ((g.n[1] + PTY - 1) / PTY);
    int chunk = g.n[2];
    while (chunk > 32 && tiles * ((g.n[2] + chunk - 1) / chunk) < (long long)sm_count() * 12) chunk = (chunk + 1) / 2;
    return chunk;
}

template <int STAGE, int NDIM>
inline void set_attr()
{
    static_assert(sizeof(Smem<STAGE>) <= 227 * 1024, "tile does not fit the shared memory of one SM");
    cudaFuncSetAttribute(stage_pair<STAGE, NDIM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(Smem<STAGE>));
    cudaFuncSetAttribute(stage_pair<STAGE, NDIM>, cudaFuncAttributePreferredSharedMemoryCarveout,
                         (int)cudaSharedmemCarveoutMaxShared);
}

inline void configure()
{
    set_attr<1, 2>();
    set_attr<2, 2>();
    set_attr<1, 3>();
    set_attr<2, 3>();
}

template <int STAGE, int NDIM>
inline void launch_impl(const double* Uin, const double* U0, double* Uout, const Grid& g, Ctrl* ctrl, int zchunk,
                        cudaStream_t stream)
{
    dim3 grid((g.n[0] + PTX - 1) / PTX, (g.n[1] + PTY - 1) / PTY, (NDIM == 3) ? (g.n[2] + zchunk - 1) / zchunk : 1);
    stage_pair<STAGE, NDIM><<<grid, NTHREADS, sizeof(Smem<STAGE>), stream>>>(Uin, U0, Uout, g, ctrl, zchunk);
}

inline void launch_stage(int stage, const double* Uin, const double* U0, double* Uout, const Grid& g, Ctrl* ctrl,
                         int zchunk, cudaStream_t stream)
{
    if (g.active[2]) {
        if (stage == 1) launch_impl<1, 3>(Uin, U0, Uout, g, ctrl, zchunk, stream);
        else            launch_impl<2, 3>(Uin, U0, Uout, g, ctrl, zchunk, stream);
    } else {
        if (stage == 1) launch_impl<1, 2>(Uin, U0, Uout, g, ctrl, zchunk, stream);
        else            launch_impl<2, 2>(Uin, U0, Uout, g, ctrl, zchunk, stream);
    }
}

}  // namespace pr
}  // namespace kh
