// kh_vanleer.cuh -- the memory-optimised second-order van Leer integrator of Sec. 3.3.
//
// "This integrator can store the prediction substep results in the space for primitive variables with reduced
//  precision, since the van Leer integrator does not directly use the prediction step in the final results.  Such
//  approach saves up to ~1/3 of the device memory for hydrodynamics, while keeping the conservation law up to the
//  full machine accuracy."
//
// The paper prints no formulas; reading S15, the same as the oracle's orc_step_vl:
//     predictor   W^{n+1/2} = prim( U^n + (dt/2) L_1(U^n) )     L_1: piecewise-constant face states + HLLC
//     corrector   U^{n+1}   = U^n + dt L_2(W^{n+1/2})           L_2: minmod PLM (Eq. 3) + HLLC (Eq. 4-5)
// Device memory: U (5 fp64 per cell) + W^{n+1/2} (5 float_t per cell: 20 B in mixed precision) instead of the two
// fp64 copies of the Heun path -- 60 instead of 80 B per cell.  Algorithmic HBM traffic per step:
// predictor 40 B read + 20 B written, corrector 20 + 40 B read + 40 B written = 160 B per cell (Heun: 200).
//
// First version: one thread per cell with the stencil read from global memory (the structure of kh_simple.cuh; any
// combination of active axes).  Each face is evaluated by both cells that share it through the same non-inlined
// function with the same inputs, so the fp64 contributions cancel bit for bit.
#pragma once
#include "kh_device.cuh"
#include "kh_simple.cuh"

namespace kh {
namespace vl {

// ---- predictor: first-order flux through the low face of cell (ci,cj,ck) along axis d ----------------------
template <typename T>
__device__ __noinline__ void face_flux_const(const double* __restrict__ U, const Grid& g, int ci, int cj, int ck,
                                             int d, T Fout[5], double pfl)
{
    const double gm1 = g.gamma - 1.0;
    const GasConst<T> gc(g.gamma, 0.0);
    int cl[3] = {ci, cj, ck};
    cl[d] -= 1;
    const Prim<T> L = load_prim<T>(U, g, cl[0], cl[1], cl[2], d, gm1, nullptr, pfl);
    const Prim<T> R = load_prim<T>(U, g, ci, cj, ck, d, gm1, nullptr, pfl);
    T F[5];
    hllc(L, R, gc, F);
    Fout[0] = F[0];
    Fout[1 + d] = F[1];
    Fout[1 + (d + 1) % 3] = F[2];
    Fout[1 + (d + 2) % 3] = F[3];
    Fout[4] = F[4];
}

// W^{n+1/2} = prim(U^n + dt/2 L_1(U^n)), stored as float_t primitives (rho, p, vx, vy, vz), SoA [5][N].
template <typename T>
__global__ void __launch_bounds__(128) predict(const double* __restrict__ U, T* __restrict__ Wh, Grid g, Ctrl* ctrl)
{
    const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const double dt = ctrl->dt;
    const double pfl = mixed_pressure_floor<T, double>(ctrl);   // the floor of the TMA predictor in mixed precision
    int hits = 0;
    if (c < g.N && dt > 0.0) {
        const int i = (int)(c % g.n[0]);
        const int j = (int)((c / g.n[0]) % g.n[1]);
        const int k = (int)(c / ((long long)g.n[0] * g.n[1]));
        double dU[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
        for (int d = 0; d < 3; d++) {
            if (!g.active[d]) continue;
            const double hdtdx = 0.5 * dt * g.inv_dx[d];
            for (int side = 0; side < 2; side++) {
                int cc[3] = {i, j, k};
                cc[d] += side;
                T F[5];
                face_flux_const<T>(U, g, cc[0], cc[1], cc[2], d, F, pfl);
                const double sgn = side ? -hdtdx : hdtdx;
#pragma unroll
                for (int m = 0; m < 5; m++) dU[m] += sgn * (double)F[m];
            }
        }
        const double gm1 = g.gamma - 1.0;
        double p, vx, vy, vz, rho;
        // floor statistics as in the Heun stages: the recovery of the own cell of U^n, then that of U^{n+1/2}
        hits = cons_to_prim(U[c], U[g.N + c], U[2 * g.N + c], U[3 * g.N + c], U[4 * g.N + c], gm1, p, vx, vy, vz, rho, pfl);
        hits += cons_to_prim(U[c] + dU[0], U[g.N + c] + dU[1], U[2 * g.N + c] + dU[2], U[3 * g.N + c] + dU[3],
                             U[4 * g.N + c] + dU[4], gm1, p, vx, vy, vz, rho);   // W^{n+1/2} is stored with the plain
        // 1e-30 floor, as the TMA predictor stores it (kh_tma.cuh, MODE 1: recover(..., pref = 0))
        Wh[c] = T(rho);
        Wh[g.N + c] = T(p);
        Wh[2 * g.N + c] = T(vx);
        Wh[3 * g.N + c] = T(vy);
        Wh[4 * g.N + c] = T(vz);
    }
    if (hits) atomicAdd(&ctrl->floor_hits, (unsigned long long)hits);
}

// ---- corrector -------------------------------------------------------------------------------------------
// Primitive state of the (possibly ghost) cell at (ci,cj,ck) read from W^{n+1/2}, boundary rules of Sec. 3.1.1
// applied to the primitives, in the frame whose normal is axis d.
template <typename T>
__device__ __forceinline__ Prim<T> load_half(const T* __restrict__ Wh, const Grid& g, int ci, int cj, int ck, int d)
{
    int rx, ry, rz;
    const int si = g.active[0] ? bc_source(ci, g.n[0], g.bc[0], g.bc[1], rx) : (rx = VN_KEEP, 0);
    const int sj = g.active[1] ? bc_source(cj, g.n[1], g.bc[2], g.bc[3], ry) : (ry = VN_KEEP, 0);
    const int sk = g.active[2] ? bc_source(ck, g.n[2], g.bc[4], g.bc[5], rz) : (rz = VN_KEEP, 0);
    const long long c = cell_index(g, si, sj, sk);
    const T vv[3] = {apply_vn_rule(Wh[2 * g.N + c], rx), apply_vn_rule(Wh[3 * g.N + c], ry),
                     apply_vn_rule(Wh[4 * g.N + c], rz)};
    Prim<T> W;
    W.r = Wh[c];
    W.p = Wh[g.N + c];
    W.u = vv[d];
    W.v = vv[(d + 1) % 3];
    W.w = vv[(d + 2) % 3];
    return W;
}

template <typename T>
__device__ __noinline__ void face_flux_half(const T* __restrict__ Wh, const Grid& g, int ci, int cj, int ck, int d,
                                            T Fout[5])
{
    const GasConst<T> gc(g.gamma, 0.0);
    Prim<T> W[4];
#pragma unroll
    for (int s = 0; s < 4; s++) {
        int cc[3] = {ci, cj, ck};
        cc[d] += s - 2;
        W[s] = load_half<T>(Wh, g, cc[0], cc[1], cc[2], d);
    }
    Prim<T> L, R;
    L.r = W[1].r + half_slope(W[0].r, W[1].r, W[2].r);
    L.p = W[1].p + half_slope(W[0].p, W[1].p, W[2].p);
    L.u = W[1].u + half_slope(W[0].u, W[1].u, W[2].u);
    L.v = W[1].v + half_slope(W[0].v, W[1].v, W[2].v);
    L.w = W[1].w + half_slope(W[0].w, W[1].w, W[2].w);
    R.r = W[2].r - half_slope(W[1].r, W[2].r, W[3].r);
    R.p = W[2].p - half_slope(W[1].p, W[2].p, W[3].p);
    R.u = W[2].u - half_slope(W[1].u, W[2].u, W[3].u);
    R.v = W[2].v - half_slope(W[1].v, W[2].v, W[3].v);
    R.w = W[2].w - half_slope(W[1].w, W[2].w, W[3].w);
    T F[5];
    hllc(L, R, gc, F);
    Fout[0] = F[0];
    Fout[1 + d] = F[1];
    Fout[1 + (d + 1) % 3] = F[2];
    Fout[1 + (d + 2) % 3] = F[3];
    Fout[4] = F[4];
}

// U^{n+1} = U^n + dt L_2(W^{n+1/2}), in place (a thread touches only its own cell of U), fp64 accumulation
// (PAPER.md:232-238); CFL rate of the new state for the next step.
template <typename T>
__global__ void __launch_bounds__(128) correct(const T* __restrict__ Wh, double* U, Grid g, Ctrl* ctrl)
{
    __shared__ double red[32];
    const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const double dt = ctrl->dt;
    double rate = 0.0;
    if (c < g.N && dt > 0.0) {
        const int i = (int)(c % g.n[0]);
        const int j = (int)((c / g.n[0]) % g.n[1]);
        const int k = (int)(c / ((long long)g.n[0] * g.n[1]));
        double dU[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
        for (int d = 0; d < 3; d++) {
            if (!g.active[d]) continue;
            const double dtdx = dt * g.inv_dx[d];
            for (int side = 0; side < 2; side++) {
                int cc[3] = {i, j, k};
                cc[d] += side;
                T F[5];
                face_flux_half<T>(Wh, g, cc[0], cc[1], cc[2], d, F);
                const double sgn = side ? -dtdx : dtdx;
#pragma unroll
                for (int m = 0; m < 5; m++) dU[m] += sgn * (double)F[m];
            }
        }
        double Un[5];
#pragma unroll
        for (int m = 0; m < 5; m++) {
            Un[m] = U[m * g.N + c] + dU[m];
            U[m * g.N + c] = Un[m];
        }
        rate = (double)cfl_rate_from_cons<T>(Un, CflConst<T>(g));
        if (!(rate == rate)) rate = __longlong_as_double(0x7ff0000000000000LL);
    }
    block_atomic_max_nonneg(rate, &ctrl->rate_bits, red);
}

template <typename T>
inline void launch_step(double* U, void* Wh, const Grid& g, Ctrl* ctrl, cudaStream_t stream, int which)
{
    const int threads = 128;
    const unsigned blocks = (unsigned)((g.N + threads - 1) / threads);
    if (which == 1) predict<T><<<blocks, threads, 0, stream>>>(U, (T*)Wh, g, ctrl);
    else            correct<T><<<blocks, threads, 0, stream>>>((const T*)Wh, U, g, ctrl);
}

}  // namespace vl
}  // namespace kh
