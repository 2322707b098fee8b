// kh_simple.cuh -- KRATOS_KERNEL_SIMPLE: one thread per cell, stencil read from global memory.
//
// The correctness anchor and the general path (any combination of active axes, any extent
// >= 4).  One fused kernel per Heun stage: boundary rules applied while the stencil is
// loaded, primitive recovery, PLM-minmod, HLLC at the cell's 2*ndim faces, fp64 flux-difference
// update, and in stage 2 the CFL rate of the new state.  Each face is evaluated by both cells
// that share it through the SAME non-inlined function with the same inputs, so the two
// contributions cancel bit for bit (conservation to float2_t accuracy).
#pragma once
#include "kh_device.cuh"

namespace kh {

// Primitive state of the (possibly ghost) cell at coordinates c[3], in the frame whose normal
// is axis d: u = v_d, v = v_{d+1}, w = v_{d+2} (cyclic).  Counts floor hits only for cells the
// caller owns (count = true).  S = float2_t, the type the conserved state is stored in (double; float in the
// all-fp32 "Single" mode, where the recovery runs in fp32 as well).
template <typename T, typename S = double>
__device__ __forceinline__ Prim<T> load_prim(const S* __restrict__ U, const Grid& g, int ci, int cj, int ck,
                                             int d, S gm1, int* hits, S pfl = S(KH_P_FLOOR))
{
    int rx, ry, rz;
    const int si = g.active[0] ? bc_source(ci, g.n[0], g.bc[0], g.bc[1], rx) : (rx = VN_KEEP, 0);
    const int sj = g.active[1] ? bc_source(cj, g.n[1], g.bc[2], g.bc[3], ry) : (ry = VN_KEEP, 0);
    const int sk = g.active[2] ? bc_source(ck, g.n[2], g.bc[4], g.bc[5], rz) : (rz = VN_KEEP, 0);
    const long long c = cell_index(g, si, sj, sk);
    S rho, p, vx, vy, vz;
    const int h = cons_to_prim(U[c], U[g.N + c], U[2 * g.N + c], U[3 * g.N + c], U[4 * g.N + c], gm1, p, vx, vy,
                               vz, rho, pfl);
    if (hits) *hits += h;
    vx = apply_vn_rule(vx, rx);
    vy = apply_vn_rule(vy, ry);
    vz = apply_vn_rule(vz, rz);
    Prim<T> W;
    W.r = T(rho);
    W.p = T(p);
    const S vv[3] = {vx, vy, vz};
    W.u = T(vv[d]);
    W.v = T(vv[(d + 1) % 3]);
    W.w = T(vv[(d + 2) % 3]);
    return W;
}

// Flux through the low face (coordinate c_d - 1/2) of cell (ci,cj,ck) along axis d, returned in
// conserved-field order (rho, m_x, m_y, m_z, eps).
template <typename T, typename S = double>
__device__ __noinline__ void face_flux_global(const S* __restrict__ U, const Grid& g, int ci, int cj, int ck,
                                              int d, T Fout[5], S pfl = S(KH_P_FLOOR))
{
    const S gm1 = S(g.gamma - 1.0);
    const GasConst<T> gc(g.gamma, 0.0);
    int c[3] = {ci, cj, ck};
    Prim<T> W[4];
#pragma unroll
    for (int s = 0; s < 4; s++) {
        int cc[3] = {c[0], c[1], c[2]};
        cc[d] += s - 2;
        W[s] = load_prim<T, S>(U, g, cc[0], cc[1], cc[2], d, gm1, nullptr, pfl);
    }
    Prim<T> L, R;
    // left state: cell c-1 plus its half slope; right state: cell c minus its half slope
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

// One Heun stage.  STAGE 1: Uout = Uin + dt L(Uin).
// STAGE 2: Uout = 1/2 U0 + 1/2 (Uin + dt L(Uin)) (Uout may alias U0), plus the CFL rate of Uout.
template <typename T, int STAGE, typename S = double>
__global__ void __launch_bounds__(128) stage_simple(const S* __restrict__ Uin, const S* U0, S* Uout,
                                                    Grid g, Ctrl* ctrl)
{
    __shared__ double red[32];
    const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const double dt = ctrl->dt;
    const S pfl = mixed_pressure_floor<T, S>(ctrl);
    double rate = 0.0;
    int hits = 0;
    if (c < g.N && dt > 0.0) {
        const int i = (int)(c % g.n[0]);
        const int j = (int)((c / g.n[0]) % g.n[1]);
        const int k = (int)(c / ((long long)g.n[0] * g.n[1]));
        S dU[5] = {S(0), S(0), S(0), S(0), S(0)};   // float2_t accumulation
        for (int d = 0; d < 3; d++) {
            if (!g.active[d]) continue;
            const S dtdx = S(dt * g.inv_dx[d]);
            for (int side = 0; side < 2; side++) {
                int cc[3] = {i, j, k};
                cc[d] += side;
                T F[5];
                face_flux_global<T, S>(Uin, g, cc[0], cc[1], cc[2], d, F, pfl);
                const S sgn = side ? -dtdx : dtdx;
#pragma unroll
                for (int m = 0; m < 5; m++) dU[m] = fma_(sgn, (S)F[m], dU[m]);
            }
        }
        // floor statistics: count the primitive recovery of this thread's own cell once per stage
        {
            S p, vx, vy, vz, rho;
            hits = cons_to_prim(Uin[c], Uin[g.N + c], Uin[2 * g.N + c], Uin[3 * g.N + c], Uin[4 * g.N + c],
                                S(g.gamma - 1.0), p, vx, vy, vz, rho, pfl);
        }
        S Un[5];
#pragma unroll
        for (int m = 0; m < 5; m++) {
            const S u = add_(Uin[m * g.N + c], dU[m]);
            Un[m] = (STAGE == 1) ? u : fma_(S(0.5), U0[m * g.N + c], mul_(S(0.5), u));
            Uout[m * g.N + c] = Un[m];
        }
        if (STAGE == 2) {
            rate = (double)cfl_rate_from_cons<T, S>(Un, CflConst<T>(g));
            if (!(rate == rate)) rate = __longlong_as_double(0x7ff0000000000000LL);
        }
    }
    if (hits) atomicAdd(&ctrl->floor_hits, (unsigned long long)hits);
    if (STAGE == 2) block_atomic_max_nonneg(rate, &ctrl->rate_bits, red);
}

}  // namespace kh
