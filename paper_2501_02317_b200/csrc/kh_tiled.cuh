// kh_tiled.cuh -- KRATOS_KERNEL_TILED: the fused Heun-stage kernel for blocks with active x and y.
//
// One thread block owns a TX x TY tile of cells in the x-y plane and marches through a slab of
// z-planes (3D) or handles a single plane (2D).  Per plane and per stage each cell's conserved state
// is fetched from HBM once (cp.async straight into a shared-memory ring, no register staging),
// converted to primitives once, every limited slope is evaluated once and every face flux once:
//   * z direction: a thread keeps the primitives of its own column (planes k, k+1, k+2), the limited
//     half-slope of plane k and the (fp64) flux through face k-1/2 in registers;
//   * x and y directions: the plane's primitives (tile + 2-cell halo, boundary rules applied on load)
//     sit in shared memory; a thread computes the x- and y-slopes of its cell, publishes the left
//     face states q_L = q + slope/2 of its high faces, and evaluates the fluxes of its low faces from
//     its neighbour's q_L and its own q_R; halo threads publish the states the tile edges need and two
//     warps evaluate the tile's high-edge faces; fluxes are exchanged through shared memory.
// The three in-plane phases (tile fill, slopes, fluxes -> update) are software-pipelined over
// consecutive planes so that one iteration needs two block barriers:
//       fill(k+1) | barrier | flux(k), slopes(k+1), z-face(k+1/2) | barrier | update(k)
// The update is done in fp64 from the raw fp64 state still resident in the shared ring
// (PAPER.md:232-238), stage 2 applies the Heun average and reduces the CFL rate of the
// new state, so no separate pass over memory is needed for the time step.
//
// Bit-identical fluxes across tile and slab seams (conservation to float2_t accuracy): a face shared by
// two tiles is evaluated by both thread blocks (as an "edge" face by one, as an own low face by the
// other), and likewise the face between two slabs and the slopes of halo cells.  All of that arithmetic
// (half_slope, the face states, hllc) is written with explicitly rounded operations (add_/mul_/fma_),
// which the compiler may neither contract nor re-associate, so every copy gives the same bits.
#pragma once
#include <cuda_pipeline_primitives.h>

#include "kh_device.cuh"

namespace kh {

constexpr int TX = 32;

// Tile height and resident blocks per SM.  Two independent blocks per SM (mixed precision) keep the
// pipes busy across each other's barriers: while one block converts fluxes (XU pipe) the other solves
// Riemann problems (FMA/ALU pipes).
#ifndef KH_TY_F32
#define KH_TY_F32 16  // tile height, mixed precision
#endif
#ifndef KH_BPS_F32
#define KH_BPS_F32 1  // resident blocks per SM, mixed precision
#endif
template <typename T>
struct TileShape {
    static constexpr int TY = (sizeof(T) == 4) ? KH_TY_F32 : 8;
    static constexpr int BLOCKS_PER_SM = (sizeof(T) == 4) ? KH_BPS_F32 : 1;
};

// roles of the warps (one warp per tile row; TY >= 8)
constexpr int WARP_EDGE_Y = 6;  // evaluates the TX faces on the tile's high y edge
constexpr int WARP_EDGE_X = 7;  // evaluates the TY faces on the tile's high x edge

template <typename T, int TY, int STAGE, int NDIM>
struct TileSmem {
    static constexpr int NRING = 4 * TX + 4 * TY;
    static constexpr int NSLOT = (NDIM == 3) ? 4 : 1;
    static constexpr int NS2 = (NDIM == 3) ? 2 : 1;
    double Uraw[NSLOT][5][TY][TX];                         // raw fp64 state of the thread's own cell, planes k..k+3
    double U0raw[5][(STAGE == 2) ? TY : 1][TX];             // U0 of the plane being updated (Heun average)
    double Rraw[NS2][5][NRING];                            // raw state of the halo ring
    T Wt[5][TY + 4][TX + 4];                               // primitives of one plane, tile + halo
    T QLx[NS2][5][TY][TX + 1];                             // left states at x faces a = 0..TX (from cell a-1)
    T QLy[NS2][5][TY + 1][TX];                             // left states at y faces b = 0..TY (from cell b-1)
    T QRxe[NS2][5][TY];                                    // right state at the high x edge (from halo column TX)
    T QRye[NS2][5][TX];                                    // right state at the high y edge (from halo row TY)
    T Fx[5][TY][TX + 1];                                   // x-face fluxes, conserved-field order
    T Fy[5][TY + 1][TX];                                   // y-face fluxes
    double red[32];
    unsigned long long mbar;                               // split-phase barrier between flux and update phases
};

__device__ __forceinline__ void cp_async8(void* smem_dst, const void* gmem_src)
{
    __pipeline_memcpy_async(smem_dst, gmem_src, 8);
}

// raw conserved values -> primitives in the global frame (rho, p - p_ref, vx, vy, vz), boundary rules on v.
// Mixed precision: the reciprocal of rho is MUFU.RCP64H + one Newton step (2^-40, far below fp32
// rounding of the result); all-fp64: IEEE division.
template <typename T>
__device__ __forceinline__ int raw_to_prim(const double u[5], double gm1, double pref, int rx, int ry, int rz, T W[5])
{
    double rho = u[0];
    const bool lo_r = rho < KH_RHO_FLOOR;
    rho = lo_r ? KH_RHO_FLOOR : rho;
    double ir;
    if (sizeof(T) == 4) {
        asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(ir) : "d"(rho));
        ir = fma(ir, fma(-rho, ir, 1.0), ir);
    } else {
        ir = 1.0 / rho;
    }
    double vx = u[1] * ir, vy = u[2] * ir, vz = u[3] * ir;
    const double ekin = 0.5 * (u[1] * vx + u[2] * vy + u[3] * vz);
    double p = gm1 * (u[4] - ekin);
    const double pfl = fmax(KH_P_FLOOR, pref * 0x1p-22);   // see pr::recover (kh_pair.cuh)
    const bool lo_p = p < pfl;
    p = lo_p ? pfl : p;
    if (rx | ry | rz) {
        vx = apply_vn_rule(vx, rx);
        vy = apply_vn_rule(vy, ry);
        vz = apply_vn_rule(vz, rz);
    }
    W[0] = T(rho);
    W[1] = T(p - pref);
    W[2] = T(vx);
    W[3] = T(vy);
    W[4] = T(vz);
    return (int)lo_r + (int)lo_p;
}

// HLLC flux from face states given as arrays (rho, p - p_ref, vx, vy, vz) with the normal along axis
// DIR; result in conserved-field order, the normal-momentum flux reduced by p_ref.
template <typename T, int DIR>
__device__ __forceinline__ void face_flux(const T qL[5], const T qR[5], const GasConst<T>& gc, T Fo[5])
{
    constexpr int iu = 2 + DIR, iv = 2 + (DIR + 1) % 3, iw = 2 + (DIR + 2) % 3;
    Prim<T> L, R;
    L.r = qL[0]; L.p = qL[1]; L.u = qL[iu]; L.v = qL[iv]; L.w = qL[iw];
    R.r = qR[0]; R.p = qR[1]; R.u = qR[iu]; R.v = qR[iv]; R.w = qR[iw];
    T F[5];
    hllc(L, R, gc, F);
    Fo[0] = F[0];
    Fo[iu - 1] = F[1];
    Fo[iv - 1] = F[2];
    Fo[iw - 1] = F[3];
    Fo[4] = F[4];
}

template <typename T, int STAGE, int NDIM>
__global__ void __launch_bounds__(TX * TileShape<T>::TY, TileShape<T>::BLOCKS_PER_SM)
stage_tiled(const double* __restrict__ Uin, const double* U0, double* Uout, Grid g, Ctrl* ctrl, int zchunk)
{
    constexpr int TY = TileShape<T>::TY;
    static_assert(TY >= 8, "warp roles need at least 8 warps");
    using Smem = TileSmem<T, TY, STAGE, NDIM>;
    // element strides inside the shared arrays (compile-time: every access is base + immediate)
    constexpr int WP = TX + 4, WF = (TY + 4) * WP;             // Wt: row pitch, field stride
    constexpr int QXF = TY * (TX + 1), QXS = 5 * QXF;          // QLx: field, slot
    constexpr int QYF = (TY + 1) * TX, QYS = 5 * QYF;          // QLy
    constexpr int FXF = TY * (TX + 1), FYF = (TY + 1) * TX;    // Fx, Fy field strides
    constexpr int URF = TY * TX, URS = 5 * URF;                // Uraw / U0raw: field, slot
    constexpr int NRING = Smem::NRING;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Smem& sm = *reinterpret_cast<Smem*>(smem_raw);

    const double dt = ctrl->dt;
    if (!(dt > 0.0)) return;  // a step clipped to zero length (run_until past t_end) does nothing
    const double pref_d = (sizeof(T) == 4) ? ctrl->p_ref : 0.0;

    const int tx = threadIdx.x, ty = threadIdx.y;
    const int warp = ty, lane = tx;
    const int nx = g.n[0], ny = g.n[1], nz = g.n[2];
    const int i = blockIdx.x * TX + tx, j = blockIdx.y * TY + ty;
    const bool inb = (i < nx) && (j < ny);
    const int kbeg = (NDIM == 3) ? blockIdx.z * zchunk : 0;
    const int kend = (NDIM == 3) ? min(kbeg + zchunk, nz) : 1;
    const double gm1 = g.gamma - 1.0;
    const GasConst<T> gc(g.gamma, pref_d);
    const CflConst<T> cc(g);
    const long long N = g.N;
    const long long pl = (long long)nx * ny;

    // own cell: source column and boundary rules in x, y (identity except on ragged edge tiles)
    int rx, ry;
    const int si = bc_source(i, nx, g.bc[0], g.bc[1], rx);
    const int sj = bc_source(j, ny, g.bc[2], g.bc[3], ry);
    const double* const own_src = Uin + ((long long)sj * nx + si);
    const long long own_cell = (long long)j * nx + i;  // valid when inb

    // per-thread bases into the shared arrays
    T* const wt_own = &sm.Wt[0][ty + 2][tx + 2];
    T* const qlx0 = &sm.QLx[0][0][ty][tx];   // left state of the own low x face; the high face is +1
    T* const qly0 = &sm.QLy[0][0][ty][tx];   // left state of the own low y face; the high face is +TX
    T* const fx0 = &sm.Fx[0][ty][tx];
    T* const fy0 = &sm.Fy[0][ty][tx];
    double* const ur0 = &sm.Uraw[0][0][ty][tx];
    double* const u00 = &sm.U0raw[0][(STAGE == 2) ? ty : 0][tx];

    // halo ring, six warp-uniform groups: rows -2, -1, TY, TY+1 (warps 0..3), columns {-2,-1} (warp 4),
    // columns {TX, TX+1} (warp 5).  Rows -1, TY and columns -1, TX also publish a face state:
    //   q_L = q + h into QLx[.][row][0] / QLy[.][0][col],   q_R = q - h into QRxe[.][row] / QRye[.][col].
    bool ring = false, ring_pub = false;
    int ring_slot = 0, rrx = 0, rry = 0;
    int r_ds = 1;              // stride in Wt along the direction of the face the ring cell feeds
    int r_dstf = 0, r_dsts = 0;  // field / slot stride of the published state
    T r_sign = T(1);
    T* wt_ring = wt_own;
    T* r_dst = qlx0;
    const double* ring_src = Uin;
    {
        int ra = 0, rb = 0;
        if (warp < 4) {
            const int row = (warp < 2) ? warp - 2 : TY + warp - 2;
            ring = true;
            ring_slot = warp * TX + lane;
            ra = lane + 2;
            rb = row + 2;
            if (warp == 1) { ring_pub = true; r_ds = WP; r_dst = &sm.QLy[0][0][0][lane]; r_dstf = QYF; r_dsts = QYS; }
            if (warp == 2) { ring_pub = true; r_ds = WP; r_dst = &sm.QRye[0][0][lane]; r_dstf = TX; r_dsts = 5 * TX; r_sign = T(-1); }
        } else if (warp < 6 && lane < 2 * TY) {
            const int q = lane / TY, row = lane % TY;
            const int col = (warp == 4) ? q - 2 : TX + q;
            ring = true;
            ring_slot = 4 * TX + (warp - 4) * 2 * TY + lane;
            ra = col + 2;
            rb = row + 2;
            if (warp == 4 && q == 1) { ring_pub = true; r_dst = &sm.QLx[0][0][row][0]; r_dstf = QXF; r_dsts = QXS; }
            if (warp == 5 && q == 0) { ring_pub = true; r_dst = &sm.QRxe[0][0][row]; r_dstf = TY; r_dsts = 5 * TY; r_sign = T(-1); }
        }
        if (ring) {
            const int gi = blockIdx.x * TX + ra - 2, gj = blockIdx.y * TY + rb - 2;
            const int ri = bc_source(gi, nx, g.bc[0], g.bc[1], rrx);
            const int rj = bc_source(gj, ny, g.bc[2], g.bc[3], rry);
            ring_src = Uin + ((long long)rj * nx + ri);
            wt_ring = &sm.Wt[0][rb][ra];
        }
    }
    double* const rr0 = &sm.Rraw[0][0][ring_slot];
    const bool edge_x = (warp == WARP_EDGE_X) && (lane < TY);  // face (a = TX, b = lane)
    const bool edge_y = (warp == WARP_EDGE_Y);                 // face (a = lane, b = TY)

    const double dtdx = dt * g.inv_dx[0], dtdy = dt * g.inv_dx[1], dtdz = dt * g.inv_dx[2];
    int hits = 0;
    T rate = T(0);

    // ---- asynchronous fetches (global -> shared, 8 bytes per field) ----
    auto fetch_own = [&](int kk) {
        int rz;
        const int sk = (NDIM == 3) ? bc_source(kk, nz, g.bc[4], g.bc[5], rz) : 0;
        const double* src = own_src + sk * pl;
        double* dst = ur0 + ((NDIM == 3) ? (kk & 3) * URS : 0);
#pragma unroll
        for (int f = 0; f < 5; f++) cp_async8(dst + f * URF, src + f * N);
    };
    auto fetch_ring = [&](int kk) {  // kk in [kbeg, kend): an interior plane
        if (!ring) return;
        const double* src = ring_src + (long long)kk * pl;
        double* dst = rr0 + ((NDIM == 3) ? (kk & 1) * (5 * NRING) : 0);
#pragma unroll
        for (int f = 0; f < 5; f++) cp_async8(dst + f * NRING, src + f * N);
    };
    auto fetch_u0 = [&](int kk) {
        if (STAGE != 2 || !inb) return;
        const double* src = U0 + ((long long)kk * pl + own_cell);
#pragma unroll
        for (int f = 0; f < 5; f++) cp_async8(u00 + f * URF, src + f * N);
    };
    auto convert_own = [&](int kk, T W[5], bool count) {
        int rz = VN_KEEP;
        if (NDIM == 3) (void)bc_source(kk, nz, g.bc[4], g.bc[5], rz);
        const double* s = ur0 + ((NDIM == 3) ? (kk & 3) * URS : 0);
        double u[5];
#pragma unroll
        for (int f = 0; f < 5; f++) u[f] = s[f * URF];
        const int h = raw_to_prim<T>(u, gm1, pref_d, rx, ry, rz, W);
        if (count && inb) hits += h;
    };

    // ---- phase 1: primitives of plane kp (own cell from registers, halo from the raw ring) -> tile ----
    T Wring[5] = {T(0), T(0), T(0), T(0), T(0)};
    auto fill_tile = [&](int kp, const T Wown[5]) {
#pragma unroll
        for (int f = 0; f < 5; f++) wt_own[f * WF] = Wown[f];
        if (ring) {
            const double* s = rr0 + ((NDIM == 3) ? (kp & 1) * (5 * NRING) : 0);
            double u[5];
#pragma unroll
            for (int f = 0; f < 5; f++) u[f] = s[f * NRING];
            (void)raw_to_prim<T>(u, gm1, pref_d, rrx, rry, VN_KEEP, Wring);
#pragma unroll
            for (int f = 0; f < 5; f++) wt_ring[f * WF] = Wring[f];
        }
    };

    // ---- phase 2a: limited slopes of plane kp; publish the left states of the own high faces ----
    auto slopes = [&](int kp, const T Wown[5], T hsx[5], T hsy[5]) {
        const int qs = (NDIM == 3) ? (kp & 1) : 0;
        T* const qx = qlx0 + qs * QXS + 1;
        T* const qy = qly0 + qs * QYS + TX;
#pragma unroll
        for (int f = 0; f < 5; f++) {
            hsx[f] = half_slope(wt_own[f * WF - 1], Wown[f], wt_own[f * WF + 1]);
            qx[f * QXF] = add_(Wown[f], hsx[f]);
        }
#pragma unroll
        for (int f = 0; f < 5; f++) {
            hsy[f] = half_slope(wt_own[f * WF - WP], Wown[f], wt_own[f * WF + WP]);
            qy[f * QYF] = add_(Wown[f], hsy[f]);
        }
        if (ring_pub) {  // halo cells next to the tile: the state the tile's edge faces need
            T* const d = r_dst + qs * r_dsts;
#pragma unroll
            for (int f = 0; f < 5; f++) {
                const T h = half_slope(wt_ring[f * WF - r_ds], Wring[f], wt_ring[f * WF + r_ds]);
                d[f * r_dstf] = fma_(r_sign, h, Wring[f]);  // q + h or q - h, exactly
            }
        }
    };

    // ---- phase 2b: x and y face fluxes of plane k ----
    T Fxlo[5], Fylo[5];
    auto fluxes = [&](int k, const T W0[5], const T hsx[5], const T hsy[5]) {
        const int qs = (NDIM == 3) ? (k & 1) : 0;
        {
            const T* const ql = qlx0 + qs * QXS;
            T qL[5], qR[5];
#pragma unroll
            for (int f = 0; f < 5; f++) { qL[f] = ql[f * QXF]; qR[f] = sub_(W0[f], hsx[f]); }
            face_flux<T, 0>(qL, qR, gc, Fxlo);
#pragma unroll
            for (int f = 0; f < 5; f++) fx0[f * FXF] = Fxlo[f];
        }
        {
            const T* const ql = qly0 + qs * QYS;
            T qL[5], qR[5];
#pragma unroll
            for (int f = 0; f < 5; f++) { qL[f] = ql[f * QYF]; qR[f] = sub_(W0[f], hsy[f]); }
            face_flux<T, 1>(qL, qR, gc, Fylo);
#pragma unroll
            for (int f = 0; f < 5; f++) fy0[f * FYF] = Fylo[f];
        }
        if (edge_x) {  // the TY faces on the tile's high x edge
            const T* const ql = &sm.QLx[qs][0][lane][TX];
            const T* const qr = &sm.QRxe[qs][0][lane];
            T qL[5], qR[5], F[5];
#pragma unroll
            for (int f = 0; f < 5; f++) { qL[f] = ql[f * QXF]; qR[f] = qr[f * TY]; }
            face_flux<T, 0>(qL, qR, gc, F);
#pragma unroll
            for (int f = 0; f < 5; f++) sm.Fx[f][lane][TX] = F[f];
        }
        if (edge_y) {  // the TX faces on the tile's high y edge
            const T* const ql = &sm.QLy[qs][0][TY][lane];
            const T* const qr = &sm.QRye[qs][0][lane];
            T qL[5], qR[5], F[5];
#pragma unroll
            for (int f = 0; f < 5; f++) { qL[f] = ql[f * QYF]; qR[f] = qr[f * TX]; }
            face_flux<T, 1>(qL, qR, gc, F);
#pragma unroll
            for (int f = 0; f < 5; f++) sm.Fy[f][TY][lane] = F[f];
        }
    };

    // ---- phase 3: fp64 flux-difference update of cell (i,j,k) ----
    auto update_cell = [&](int k, const double Fzlo[5], const double Fzhi[5]) {
        if (!inb) return;
        const double* su = ur0 + ((NDIM == 3) ? (k & 3) * URS : 0);
        const double* s0 = u00;
        double* out = Uout + ((long long)k * pl + own_cell);
        double Un[5];
#pragma unroll
        for (int f = 0; f < 5; f++) {
            double dU = dtdx * ((double)Fxlo[f] - (double)fx0[f * FXF + 1]);
            dU = fma(dtdy, (double)Fylo[f] - (double)fy0[f * FYF + TX], dU);
            if (NDIM == 3) dU = fma(dtdz, Fzlo[f] - Fzhi[f], dU);
            const double u = su[f * URF] + dU;
            Un[f] = (STAGE == 1) ? u : 0.5 * s0[f * URF] + 0.5 * u;
            out[f * N] = Un[f];
        }
        if (STAGE == 2) {
            T r = cfl_rate_from_cons<T>(Un, cc);
            if (!(r == r)) r = T(__int_as_float(0x7f800000));
            rate = fmax(rate, r);
        }
    };

    if (NDIM == 2) {
        fetch_own(0);
        fetch_ring(0);
        fetch_u0(0);
        __pipeline_commit();
        __pipeline_wait_prior(0);
        T W0[5], hsx[5], hsy[5];
        convert_own(0, W0, true);
        fill_tile(0, W0);
        __syncthreads();
        slopes(0, W0, hsx, hsy);
        __syncthreads();
        fluxes(0, W0, hsx, hsy);
        __syncthreads();
        const double Fz[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
        update_cell(0, Fz, Fz);
    } else {
        // prologue: planes kbeg-2 .. kbeg+1 of the own column, halo ring of plane kbeg
        fetch_own(kbeg - 2);
        fetch_own(kbeg - 1);
        fetch_own(kbeg);
        fetch_own(kbeg + 1);
        fetch_ring(kbeg);
        __pipeline_commit();
        __pipeline_wait_prior(0);
        T W0[5], Wp1[5], Wp2[5], hs0[5], hsx[5], hsy[5];
        double Fzlo[5];
        {
            T Wm[5];
            convert_own(kbeg - 2, Wm, false);
            convert_own(kbeg - 1, W0, false);
            convert_own(kbeg, Wp1, true);
#pragma unroll
            for (int f = 0; f < 5; f++) {
                hs0[f] = half_slope(Wm[f], W0[f], Wp1[f]);
                Fzlo[f] = 0.0;
                hsx[f] = hsy[f] = T(0);
                Fxlo[f] = Fylo[f] = T(0);
            }
        }
        if (tx == 0 && ty == 0) mbar_init(&sm.mbar, TX * TY);
        __syncthreads();
        // iteration k: fill(k+1) | barrier | flux(k), slopes(k+1) | arrive | z face k+1/2 | wait | update(k).
        // k = kbeg-1 only primes the pipeline (tile and slopes of plane kbeg, low z face of the slab).
#pragma unroll 1
        for (int k = kbeg - 1; k < kend; k++) {
            // two cp.async groups per iteration, oldest first: {U0(k)} issued after update(k-1), then
            // {own(k+3), ring(k+2)}.  Here only the previous iteration's {own, ring} group must have landed.
            if (k + 3 <= kend + 1) fetch_own(k + 3);
            if (k + 2 < kend) fetch_ring(k + 2);
            __pipeline_commit();
            __pipeline_wait_prior(2);
            const bool next = k + 1 < kend;
            if (next) fill_tile(k + 1, Wp1);
            __syncthreads();
            if (k >= kbeg) fluxes(k, W0, hsx, hsy);
            if (next) slopes(k + 1, Wp1, hsx, hsy);
            // arrive now, wait after the z face: that work needs nothing from other threads
            const unsigned long long token = mbar_arrive(&sm.mbar);
            // z face k+1/2 from the register-resident column
            convert_own(k + 2, Wp2, k + 2 < kend);
            T hs1[5];
            double Fzhi[5];
            {
                T qL[5], qR[5], F[5];
#pragma unroll
                for (int f = 0; f < 5; f++) {
                    hs1[f] = half_slope(W0[f], Wp1[f], Wp2[f]);
                    qL[f] = add_(W0[f], hs0[f]);
                    qR[f] = sub_(Wp1[f], hs1[f]);
                }
                face_flux<T, 2>(qL, qR, gc, F);
#pragma unroll
                for (int f = 0; f < 5; f++) Fzhi[f] = (double)F[f];
            }
            if (STAGE == 2) __pipeline_wait_prior(1);  // U0(k) has landed (own thread's copy)
            mbar_wait(&sm.mbar, token);                // every thread's x/y fluxes of plane k are published
            if (k >= kbeg) update_cell(k, Fzlo, Fzhi);
            if (k + 1 < kend) fetch_u0(k + 1);  // single slot: only after this thread has read U0(k)
            __pipeline_commit();
#pragma unroll
            for (int f = 0; f < 5; f++) { W0[f] = Wp1[f]; Wp1[f] = Wp2[f]; hs0[f] = hs1[f]; Fzlo[f] = Fzhi[f]; }
        }
        __pipeline_wait_prior(0);
    }

    if (hits) atomicAdd(&ctrl->floor_hits, (unsigned long long)hits);
    if (STAGE == 2) {
        __syncthreads();
        block_atomic_max_nonneg((double)rate, &ctrl->rate_bits, sm.red);
    }
}

// ---------------------------------------------------------------------------------------
// host side
inline int tiled_auto_zchunk(const Grid& g)
{
    if (!g.active[2]) return 1;
    // enough thread blocks for >= ~12 waves over the SMs (148 on B200; one block per SM), slabs of >= 16 planes
    const long long tiles = (long long)((g.n[0] + TX - 1) / TX) * ((g.n[1] + KH_TY_F32 - 1) / KH_TY_F32);
    int chunk = g.n[2];
    while (chunk > 16 && tiles * ((g.n[2] + chunk - 1) / chunk) < (long long)sm_count() * KH_BPS_F32 * 12) chunk = (chunk + 1) / 2;
    return chunk;
}

template <typename T, int STAGE, int NDIM>
inline void tiled_set_attr()
{
    using S = TileSmem<T, TileShape<T>::TY, STAGE, NDIM>;
    static_assert(sizeof(S) * TileShape<T>::BLOCKS_PER_SM <= 227 * 1024 - 1024 * TileShape<T>::BLOCKS_PER_SM,
                  "tiles do not fit the shared memory of one SM");
    cudaFuncSetAttribute(stage_tiled<T, STAGE, NDIM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(S));
    cudaFuncSetAttribute(stage_tiled<T, STAGE, NDIM>, cudaFuncAttributePreferredSharedMemoryCarveout,
                         (int)cudaSharedmemCarveoutMaxShared);
}

inline void tiled_configure()
{
    tiled_set_attr<float, 1, 2>(); tiled_set_attr<float, 2, 2>();
    tiled_set_attr<float, 1, 3>(); tiled_set_attr<float, 2, 3>();
    tiled_set_attr<double, 1, 2>(); tiled_set_attr<double, 2, 2>();
    tiled_set_attr<double, 1, 3>(); tiled_set_attr<double, 2, 3>();
}

template <typename T, int STAGE, int NDIM>
inline void launch_stage_tiled_impl(const double* Uin, const double* U0, double* Uout, const Grid& g, Ctrl* ctrl,
                                    int zchunk, cudaStream_t stream)
{
    constexpr int TY = TileShape<T>::TY;
    using S = TileSmem<T, TY, STAGE, NDIM>;
    dim3 block(TX, TY, 1);
    dim3 grid((g.n[0] + TX - 1) / TX, (g.n[1] + TY - 1) / TY, (NDIM == 3) ? (g.n[2] + zchunk - 1) / zchunk : 1);
    stage_tiled<T, STAGE, NDIM><<<grid, block, sizeof(S), stream>>>(Uin, U0, Uout, g, ctrl, zchunk);
}

template <typename T>
inline void launch_stage_tiled(int stage, const double* Uin, const double* U0, double* Uout, const Grid& g,
                               Ctrl* ctrl, int zchunk, cudaStream_t stream)
{
    if (g.active[2]) {
        if (stage == 1) launch_stage_tiled_impl<T, 1, 3>(Uin, U0, Uout, g, ctrl, zchunk, stream);
        else            launch_stage_tiled_impl<T, 2, 3>(Uin, U0, Uout, g, ctrl, zchunk, stream);
    } else {
        if (stage == 1) launch_stage_tiled_impl<T, 1, 2>(Uin, U0, Uout, g, ctrl, zchunk, stream);
        else            launch_stage_tiled_impl<T, 2, 2>(Uin, U0, Uout, g, ctrl, zchunk, stream);
    }
}

}  // namespace kh
