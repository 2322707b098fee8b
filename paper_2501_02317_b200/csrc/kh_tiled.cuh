// kh_tiled.cuh -- KRATOS_KERNEL_TILED: the fused Heun-stage kernel for blocks with active x and y.
//
// One thread block owns a TX x TY tile of cells in the x-y plane and marches through a slab of
// z-planes (3D) or handles a single plane (2D).  Per plane and per stage each cell's conserved
// state is fetched from HBM once (cp.async straight into a shared-memory ring, no register
// staging), converted to primitives once, and every face flux is evaluated exactly once:
//   * z direction: each thread keeps the primitives of its own column (planes k, k+1, k+2), the
//     limited half-slope of plane k and the flux through face k-1/2 in registers;
//   * x and y directions: the plane's primitives (tile + 2-cell halo, boundary rules applied on
//     load) sit in shared memory; a thread evaluates the low x- and y-face of its cell, two
//     spare warps evaluate the tile's high-edge faces, and fluxes are exchanged through shared
//     memory.
// The update is done in fp64 from the raw fp64 state still resident in the shared ring
// (PAPER.md:232-238), stage 2 applies the Heun average and reduces the CFL rate of
// the new state so that no separate pass over memory is needed for the time step.
//
// Bit-identical fluxes across tile and slab seams (conservation to float2_t accuracy): every
// face class (x, y, z) has exactly ONE instruction sequence in the kernel -- regular and edge
// faces run through the same non-unrolled loop body, and the face below a slab is produced by the
// same loop iteration code as the face on top of the previous slab.
#pragma once
#include <cuda_pipeline_primitives.h>

#include "kh_device.cuh"

namespace kh {

constexpr int TX = 32;

template <typename T>
struct TileShape {
    static constexpr int TY = (sizeof(T) == 4) ? 16 : 8;
};

template <typename T, int TY, int STAGE, int NDIM>
struct TileSmem {
    static constexpr int NRING = 4 * TX + 4 * TY;
    static constexpr int NSLOT = (NDIM == 3) ? 4 : 1;
    double Uraw[NSLOT][5][TY][TX];                       // raw fp64 state of the thread's own cell, planes k..k+3
    double U0raw[(STAGE == 2) ? ((NDIM == 3) ? 2 : 1) : 1][5][(STAGE == 2) ? TY : 1][TX];  // U0 for the Heun average
    double Rraw[(NDIM == 3) ? 2 : 1][5][NRING];          // raw state of the halo ring
    T Wt[5][TY + 4][TX + 4];                             // primitives of the current plane, tile + halo
    T Fx[5][TY][TX + 1];                                 // x-face fluxes, conserved-field order
    T Fy[5][TY + 1][TX];                                 // y-face fluxes
    double red[32];
};

__device__ __forceinline__ void cp_async8(void* smem_dst, const void* gmem_src)
{
    __pipeline_memcpy_async(smem_dst, gmem_src, 8);
}

// raw conserved values -> primitives in the global frame (rho, p, vx, vy, vz), boundary rules on v
template <typename T>
__device__ __forceinline__ int raw_to_prim(const double u[5], double gm1, int rx, int ry, int rz, T W[5])
{
    double rho, p, vx, vy, vz;
    const int h = cons_to_prim(u[0], u[1], u[2], u[3], u[4], gm1, p, vx, vy, vz, rho);
    if (rx | ry | rz) {
        vx = apply_vn_rule(vx, rx);
        vy = apply_vn_rule(vy, ry);
        vz = apply_vn_rule(vz, rz);
    }
    W[0] = T(rho);
    W[1] = T(p);
    W[2] = T(vx);
    W[3] = T(vy);
    W[4] = T(vz);
    return h;
}

// Flux through the face between tile cells (a-1, b) and (a, b) [DIR 0] or (a, b-1) and (a, b)
// [DIR 1], tile coordinates including the 2-cell halo offset.  Output in conserved-field order.
template <typename T, int TY, int DIR, typename S>
__device__ __forceinline__ void face_flux_tile(const S& sm, int a, int b, const GasConst<T>& gc, T Fo[5])
{
    T q[5][4];
#pragma unroll
    for (int f = 0; f < 5; f++)
#pragma unroll
        for (int s = 0; s < 4; s++) q[f][s] = (DIR == 0) ? sm.Wt[f][b][a - 2 + s] : sm.Wt[f][b - 2 + s][a];
    // normal-frame slots: DIR 0: (u,v,w) = (vx,vy,vz); DIR 1: (vy,vz,vx)
    constexpr int iu = (DIR == 0) ? 2 : 3, iv = (DIR == 0) ? 3 : 4, iw = (DIR == 0) ? 4 : 2;
    Prim<T> L, R;
    L.r = q[0][1] + half_slope(q[0][0], q[0][1], q[0][2]);
    R.r = q[0][2] - half_slope(q[0][1], q[0][2], q[0][3]);
    L.p = q[1][1] + half_slope(q[1][0], q[1][1], q[1][2]);
    R.p = q[1][2] - half_slope(q[1][1], q[1][2], q[1][3]);
    L.u = q[iu][1] + half_slope(q[iu][0], q[iu][1], q[iu][2]);
    R.u = q[iu][2] - half_slope(q[iu][1], q[iu][2], q[iu][3]);
    L.v = q[iv][1] + half_slope(q[iv][0], q[iv][1], q[iv][2]);
    R.v = q[iv][2] - half_slope(q[iv][1], q[iv][2], q[iv][3]);
    L.w = q[iw][1] + half_slope(q[iw][0], q[iw][1], q[iw][2]);
    R.w = q[iw][2] - half_slope(q[iw][1], q[iw][2], q[iw][3]);
    T F[5];
    hllc(L, R, gc, F);
    Fo[0] = F[0];
    Fo[4] = F[4];
    if (DIR == 0) { Fo[1] = F[1]; Fo[2] = F[2]; Fo[3] = F[3]; }
    else          { Fo[2] = F[1]; Fo[3] = F[2]; Fo[1] = F[3]; }
}

template <typename T, int STAGE, int NDIM>
__global__ void __launch_bounds__(TX * TileShape<T>::TY, 1)
stage_tiled(const double* __restrict__ Uin, const double* U0, double* Uout, Grid g, Ctrl* ctrl, int zchunk)
{
    constexpr int TY = TileShape<T>::TY;
    constexpr int NWARP = TY;  // one warp per tile row
    using Smem = TileSmem<T, TY, STAGE, NDIM>;
    constexpr int NRING = Smem::NRING;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Smem& sm = *reinterpret_cast<Smem*>(smem_raw);

    const double dt = ctrl->dt;
    if (!(dt > 0.0)) return;  // a step clipped to zero length (run_until past t_end) does nothing

    const int tx = threadIdx.x, ty = threadIdx.y;
    const int tid = ty * TX + tx;
    const int warp = ty, lane = tx;
    const int nx = g.n[0], ny = g.n[1], nz = g.n[2];
    const int i = blockIdx.x * TX + tx, j = blockIdx.y * TY + ty;
    const bool inb = (i < nx) && (j < ny);
    const int kbeg = (NDIM == 3) ? blockIdx.z * zchunk : 0;
    const int kend = (NDIM == 3) ? min(kbeg + zchunk, nz) : 1;
    const double gm1 = g.gamma - 1.0;
    const GasConst<T> gc(g.gamma);
    const long long N = g.N;
    const long long pl = (long long)nx * ny;

    // own cell: source column and boundary rules in x, y (identity except on ragged edge tiles)
    int rx, ry;
    const int si = bc_source(i, nx, g.bc[0], g.bc[1], rx);
    const int sj = bc_source(j, ny, g.bc[2], g.bc[3], ry);
    const long long own_col = (long long)sj * nx + si;

    // ring cell handled by this thread (if any): halo rows first, then halo columns
    int ring = -1;
    if (NRING <= (NWARP / 2) * 32) {  // spread over warps {0,1,4,5,...}: scheduler quadrants 0 and 1
        if ((warp & 3) < 2) { const int r = ((warp >> 2) * 2 + (warp & 3)) * 32 + lane; if (r < NRING) ring = r; }
    } else if (tid < NRING) ring = tid;
    int ra = 0, rb = 0, rrx = 0, rry = 0;  // tile coordinates (with halo offset) and rules of the ring cell
    long long ring_col = 0;
    if (ring >= 0) {
        int col, row;
        if (ring < 4 * TX) { const int q = ring / TX; col = ring % TX; row = (q < 2) ? q - 2 : TY + q - 2; }
        else { const int rr = ring - 4 * TX; const int q = rr & 3; row = rr >> 2; col = (q < 2) ? q - 2 : TX + q - 2; }
        ra = col + 2; rb = row + 2;
        const int gi = blockIdx.x * TX + col, gj = blockIdx.y * TY + row;
        const int ri = bc_source(gi, nx, g.bc[0], g.bc[1], rrx);
        const int rj = bc_source(gj, ny, g.bc[2], g.bc[3], rry);
        ring_col = (long long)rj * nx + ri;
    }

    const double dtdx = dt * g.inv_dx[0], dtdy = dt * g.inv_dx[1], dtdz = dt * g.inv_dx[2];
    int hits = 0;
    T rate = T(0);

    // ---- asynchronous fetches (global -> shared, 8 bytes per field) ----
    auto fetch_own = [&](int kk) {
        int rz;
        const int sk = (NDIM == 3) ? bc_source(kk, nz, g.bc[4], g.bc[5], rz) : 0;
        const double* src = Uin + sk * pl + own_col;
        const int slot = (NDIM == 3) ? (kk & 3) : 0;
#pragma unroll
        for (int f = 0; f < 5; f++) cp_async8(&sm.Uraw[slot][f][ty][tx], src + f * N);
    };
    auto fetch_ring = [&](int kk) {
        if (ring < 0) return;
        const double* src = Uin + (long long)kk * pl + ring_col;  // kk in [kbeg, kend): interior plane
        const int slot = (NDIM == 3) ? (kk & 1) : 0;
#pragma unroll
        for (int f = 0; f < 5; f++) cp_async8(&sm.Rraw[slot][f][ring], src + f * N);
    };
    auto fetch_u0 = [&](int kk) {
        if (STAGE != 2 || !inb) return;
        const double* src = U0 + (long long)kk * pl + (long long)j * nx + i;
        const int slot = (NDIM == 3) ? (kk & 1) : 0;
#pragma unroll
        for (int f = 0; f < 5; f++) cp_async8(&sm.U0raw[slot][f][ty][tx], src + f * N);
    };
    auto convert_own = [&](int kk, T W[5]) {
        int rz = VN_KEEP;
        if (NDIM == 3) (void)bc_source(kk, nz, g.bc[4], g.bc[5], rz);
        const int slot = (NDIM == 3) ? (kk & 3) : 0;
        double u[5];
#pragma unroll
        for (int f = 0; f < 5; f++) u[f] = sm.Uraw[slot][f][ty][tx];
        const int h = raw_to_prim<T>(u, gm1, rx, ry, rz, W);
        if (inb && kk >= kbeg && kk < kend) hits += h;
    };

    // ---- in-plane part of plane k: tile fill, x/y face fluxes ----
    auto inplane_fluxes = [&](int k, const T W0[5]) {
#pragma unroll
        for (int f = 0; f < 5; f++) sm.Wt[f][ty + 2][tx + 2] = W0[f];
        if (ring >= 0) {
            const int slot = (NDIM == 3) ? (k & 1) : 0;
            double u[5];
#pragma unroll
            for (int f = 0; f < 5; f++) u[f] = sm.Rraw[slot][f][ring];
            T Wr[5];
            (void)raw_to_prim<T>(u, gm1, rrx, rry, VN_KEEP, Wr);
#pragma unroll
            for (int f = 0; f < 5; f++) sm.Wt[f][rb][ra] = Wr[f];
        }
        __syncthreads();
        // x faces: pass 0 = low face of the own cell; pass 1 = the tile's high edge (warp 3)
#pragma unroll 1
        for (int pass = 0; pass < 2; pass++) {
            int a = tx, b = ty;
            if (pass == 1) {
                if (warp != (3 % NWARP)) break;
                if (lane >= TY) break;
                a = TX; b = lane;
            }
            T F[5];
            face_flux_tile<T, TY, 0>(sm, a + 2, b + 2, gc, F);
#pragma unroll
            for (int f = 0; f < 5; f++) sm.Fx[f][b][a] = F[f];
        }
        // y faces: pass 1 = the tile's high edge (warp 2)
#pragma unroll 1
        for (int pass = 0; pass < 2; pass++) {
            int a = tx, b = ty;
            if (pass == 1) {
                if (warp != (2 % NWARP)) break;
                a = lane; b = TY;
            }
            T F[5];
            face_flux_tile<T, TY, 1>(sm, a + 2, b + 2, gc, F);
#pragma unroll
            for (int f = 0; f < 5; f++) sm.Fy[f][b][a] = F[f];
        }
    };

    // ---- fp64 flux-difference update of cell (i,j,k) ----
    auto update_cell = [&](int k, const T Fzlo[5], const T Fzhi[5]) {
        if (!inb) return;
        const int slot = (NDIM == 3) ? (k & 3) : 0;
        const int slot0 = (NDIM == 3) ? (k & 1) : 0;
        const long long c = (long long)k * pl + (long long)j * nx + i;
        double Un[5];
#pragma unroll
        for (int f = 0; f < 5; f++) {
            double dU = dtdx * ((double)sm.Fx[f][ty][tx] - (double)sm.Fx[f][ty][tx + 1]);
            dU += dtdy * ((double)sm.Fy[f][ty][tx] - (double)sm.Fy[f][ty + 1][tx]);
            if (NDIM == 3) dU += dtdz * ((double)Fzlo[f] - (double)Fzhi[f]);
            const double u = sm.Uraw[slot][f][ty][tx] + dU;
            Un[f] = (STAGE == 1) ? u : 0.5 * sm.U0raw[slot0][f][ty][tx] + 0.5 * u;
            Uout[f * N + c] = Un[f];
        }
        if (STAGE == 2) {
            T r = cfl_rate_from_cons<T>(Un, g);
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
        T W0[5];
        convert_own(0, W0);
        inplane_fluxes(0, W0);
        __syncthreads();
        T Fz[5] = {T(0), T(0), T(0), T(0), T(0)};
        update_cell(0, Fz, Fz);
    } else {
        // prologue: planes kbeg-2 .. kbeg+1 of the own column
        fetch_own(kbeg - 2);
        fetch_own(kbeg - 1);
        fetch_own(kbeg);
        fetch_own(kbeg + 1);
        __pipeline_commit();
        __pipeline_wait_prior(0);
        T W0[5], Wp1[5], Wp2[5], hs0[5], Fzlo[5];
        {
            T Wm[5];
            convert_own(kbeg - 2, Wm);
            convert_own(kbeg - 1, W0);
            convert_own(kbeg, Wp1);
#pragma unroll
            for (int f = 0; f < 5; f++) { hs0[f] = half_slope(Wm[f], W0[f], Wp1[f]); Fzlo[f] = T(0); }
        }
        // iteration k handles face k+1/2; k = kbeg-1 only primes the low face of the slab
#pragma unroll 1
        for (int k = kbeg - 1; k < kend; k++) {
            if (k + 3 <= kend + 1) fetch_own(k + 3);
            if (k + 1 < kend) { fetch_ring(k + 1); fetch_u0(k + 1); }
            __pipeline_commit();
            __pipeline_wait_prior(1);  // everything issued before this iteration has landed
            if (k >= kbeg) inplane_fluxes(k, W0);
            // z face k+1/2 from the register-resident column; normal frame (u,v,w) = (vz,vx,vy)
            convert_own(k + 2, Wp2);
            T hs1[5], Fzhi[5];
#pragma unroll
            for (int f = 0; f < 5; f++) hs1[f] = half_slope(W0[f], Wp1[f], Wp2[f]);
            {
                Prim<T> L, R;
                L.r = W0[0] + hs0[0]; R.r = Wp1[0] - hs1[0];
                L.p = W0[1] + hs0[1]; R.p = Wp1[1] - hs1[1];
                L.u = W0[4] + hs0[4]; R.u = Wp1[4] - hs1[4];
                L.v = W0[2] + hs0[2]; R.v = Wp1[2] - hs1[2];
                L.w = W0[3] + hs0[3]; R.w = Wp1[3] - hs1[3];
                T F[5];
                hllc(L, R, gc, F);
                Fzhi[0] = F[0]; Fzhi[3] = F[1]; Fzhi[1] = F[2]; Fzhi[2] = F[3]; Fzhi[4] = F[4];
            }
            if (k >= kbeg) {
                __syncthreads();
                update_cell(k, Fzlo, Fzhi);
            }
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
    // enough thread blocks for >= ~12 waves over 148 SMs (one block per SM), slabs of >= 16 planes
    const long long tiles = (long long)((g.n[0] + TX - 1) / TX) * ((g.n[1] + 15) / 16);
    int chunk = g.n[2];
    while (chunk > 16 && tiles * ((g.n[2] + chunk - 1) / chunk) < 148LL * 12) chunk = (chunk + 1) / 2;
    return chunk;
}

template <typename T, int STAGE, int NDIM>
inline void tiled_set_attr()
{
    using S = TileSmem<T, TileShape<T>::TY, STAGE, NDIM>;
    cudaFuncSetAttribute(stage_tiled<T, STAGE, NDIM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(S));
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
