// kh_device.cuh -- device-side building blocks of the Kratos hydro hot path (sm_100a).
//
// Everything here is templated on the working type T = float_t of the paper
// (Sec. 3.2.2): float in mixed precision, double in all-fp64 mode.
// The conserved state and its update are always double (float2_t).
//
// Notation follows the paper: primitives W = (rho, p, v), conserved
// U = (rho, m, eps), s_* the contact speed (Eq. 4), Delta s_K = s_K - u_K and
// q_K the pressure-ratio factor (Eq. 5).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace kh {

enum : int { BC_PERIODIC = 0, BC_FREE = 1, BC_OUTFLOW = 2, BC_REFLECT = 3 };
// what a boundary rule does to the normal velocity of a ghost cell
enum : int { VN_KEEP = 0, VN_NEGATE = 1, VN_MIN0 = 2, VN_MAX0 = 3 };

// Device-resident control block: time, time step and reduction targets.  Kernels read dt
// from here so that no host round trip is needed between steps (kratos_hydro_run).
struct Ctrl {
    double t;                        // current time
    double dt;                       // time step the stage kernels use
    double t_end;                    // > 0: clip dt so that t lands on t_end
    double cfl;                      // Courant number used by the dt bookkeeping kernel
    unsigned long long rate_bits;    // max over cells of sum_d (|v_d|+c)/dx_d, as double bits (>= 0)
    unsigned long long floor_hits;   // primitive floor activations (reading S6)
    long long steps;                 // steps with dt > 0 taken by run / run_until
    int nonfinite;                   // set when a dt came out non-finite
    int pad;
};

// Grid description passed by value to every kernel.
struct Grid {
    int n[3];          // nx, ny, nz
    int bc[6];         // x-lo, x-hi, y-lo, y-hi, z-lo, z-hi
    int active[3];     // extent > 1
    long long N;       // nx*ny*nz = field stride of the SoA state
    double gamma;
    double inv_dx[3];  // 1/dx_d (0 for inactive axes)
};

__device__ __forceinline__ long long cell_index(const Grid& g, int i, int j, int k)
{
    return ((long long)k * g.n[1] + j) * g.n[0] + i;
}

// Sec. 3.1.1.  Map a coordinate c in [-2, n+2) along one axis to the
// interior cell the ghost value is taken from, and say what happens to the normal velocity.
// The rules are printed for the left-x face with v_x the INWARD normal component; on a
// high-side face the inward normal is -axis, so min(v_in, 0) becomes max(v_axis, 0).
// Coordinates further out than two layers are clamped (never used by the stencil).
__device__ __forceinline__ int bc_source(int c, int n, int bc_lo, int bc_hi, int& vn_rule)
{
    vn_rule = VN_KEEP;
    if (c < 0) {
        if (bc_lo == BC_PERIODIC) return max(c + n, 0);
        if (bc_lo == BC_REFLECT) { vn_rule = VN_NEGATE; return min(-1 - c, n - 1); }
        if (bc_lo == BC_OUTFLOW) vn_rule = VN_MIN0;
        return 0;
    }
    if (c >= n) {
        if (bc_hi == BC_PERIODIC) return min(c - n, n - 1);
        if (bc_hi == BC_REFLECT) { vn_rule = VN_NEGATE; return max(2 * n - 1 - c, 0); }
        if (bc_hi == BC_OUTFLOW) vn_rule = VN_MAX0;
        return n - 1;
    }
    return c;
}

template <typename T>
__device__ __forceinline__ T apply_vn_rule(T v, int rule)
{
    if (rule == VN_NEGATE) return -v;
    if (rule == VN_MIN0) return v < T(0) ? v : T(0);
    if (rule == VN_MAX0) return v > T(0) ? v : T(0);
    return v;
}

// ---------------------------------------------------------------------------------------
// fast fp32 special functions (one MUFU each); fp64 uses IEEE division and sqrt.
__device__ __forceinline__ float rcp_(float x)
{
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ double rcp_(double x) { return 1.0 / x; }
__device__ __forceinline__ float sqrt_(float x)
{
    float r;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ double sqrt_(double x) { return sqrt(x); }
__device__ __forceinline__ float rsqrt_(float x)
{
    float r;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ double rsqrt_(double x) { return 1.0 / sqrt(x); }

// c = sqrt(gamma p / rho).  fp32: gamma p * rsqrt(gamma p rho), a single MUFU.
__device__ __forceinline__ float sound_speed(float gp, float rho) { return gp * rsqrt_(gp * rho); }
__device__ __forceinline__ double sound_speed(double gp, double rho) { return sqrt(gp / rho); }

// ---------------------------------------------------------------------------------------
// Primitive state in a face-normal frame: u normal, v and w tangential.
template <typename T>
struct Prim {
    T r, p, u, v, w;
};

#define KH_RHO_FLOOR 1e-30
#define KH_P_FLOOR 1e-30

// Sec. 3.1: (rho, m, eps) -> (rho, p, v), arithmetic in fp64 in every mode
// (reading S7: p is a difference of large terms), floors on the primitives only (S6).
// Returns the number of floor activations (0, 1 or 2).
__device__ __forceinline__ int cons_to_prim(double rho, double mx, double my, double mz, double eps,
                                            double gm1, double& p, double& vx, double& vy, double& vz,
                                            double& rho_out)
{
    int hits = 0;
    if (rho < KH_RHO_FLOOR) { rho = KH_RHO_FLOOR; hits++; }
    const double ir = 1.0 / rho;
    vx = mx * ir;
    vy = my * ir;
    vz = mz * ir;
    const double ekin = 0.5 * (mx * vx + my * vy + mz * vz);
    p = gm1 * (eps - ekin);
    if (p < KH_P_FLOOR) { p = KH_P_FLOOR; hits++; }
    rho_out = rho;
    return hits;
}

// Eq. 3, reading S2 for ab = 0.
template <typename T>
__device__ __forceinline__ T minmod(T a, T b)
{
    const T m = fmin(fabs(a), fabs(b));
    return (a * b > T(0)) ? copysign(m, a) : T(0);
}

// Half the limited undivided difference: (dx/2) * minmod((q0-qm)/dx, (qp-q0)/dx) on a uniform
// mesh (reading S8; PAPER.md:242 asks for Delta x in the denominator to keep the slope from
// being a difference of large products -- the undivided difference has that property too).
template <typename T>
__device__ __forceinline__ T half_slope(T qm, T q0, T qp)
{
    return T(0.5) * minmod(q0 - qm, qp - q0);
}

// Constants of the Riemann solver, computed once per kernel.
template <typename T>
struct GasConst {
    T gamma;   // gamma
    T g1;      // (gamma+1)/(2 gamma), Eq. 5
    T igm1;    // 1/(gamma-1)
    __device__ __forceinline__ explicit GasConst(double g)
        : gamma(T(g)), g1(T((g + 1.0) / (2.0 * g))), igm1(T(1.0 / (g - 1.0))) {}
};

// Sec. 3.2.2: HLLC flux with the subtraction-safe wave speeds of Eq. 5.
//   c_K = sqrt(gamma p_K / rho_K)
//   p_* = max(0, (p_L+p_R)/2 - (u_R-u_L)/2 * rho_bar * c_bar)                        (reading S3)
//   q_K = sqrt(1 + (gamma+1)/(2 gamma) * max(p_*/p_K - 1, 0)),  Delta s_L = -c_L q_L,  Delta s_R = +c_R q_R
//   s_* = {[p_R - rho_R u_R Ds_R] - [p_L - rho_L u_L Ds_L]} / {rho_L Ds_L - rho_R Ds_R}        (Eq. 4)
// Flux on the side K of the contact that contains x/t = 0, written in Ds_K throughout
// (an algebraically equivalent form of the star-state assembly, reading S4):
//   m_K = rho_K Ds_K,  p_*K = p_K + m_K (s_* - u_K),  phi = s_* / (s_K - s_*),
//   F_rho = phi m_K,  F_u = p_*K + F_rho s_*,  F_E = s_* [ (E_K Ds_K - p_K u_K)/(s_K - s_*) + p_*K (1 + phi) ],
//   F_v = F_rho v_K,  F_w = F_rho w_K;
// outside the fan (s_L >= 0 or s_R <= 0) the upwind physical flux.
// F = (mass, normal momentum, tangential momentum 1, tangential momentum 2, energy).
template <typename T>
__device__ __forceinline__ void hllc(const Prim<T>& L, const Prim<T>& R, const GasConst<T>& gc, T F[5])
{
    const T cL = sound_speed(gc.gamma * L.p, L.r);
    const T cR = sound_speed(gc.gamma * R.p, R.r);

    T pst = T(0.5) * (L.p + R.p) - T(0.125) * (R.u - L.u) * (L.r + R.r) * (cL + cR);
    pst = fmax(pst, T(0));

    const T qL = sqrt_(T(1) + gc.g1 * fmax(pst * rcp_(L.p) - T(1), T(0)));
    const T qR = sqrt_(T(1) + gc.g1 * fmax(pst * rcp_(R.p) - T(1), T(0)));
    const T dsL = -cL * qL;
    const T dsR = cR * qR;
    const T mL = L.r * dsL;
    const T mR = R.r * dsR;
    const T sst = ((R.p - mR * R.u) - (L.p - mL * L.u)) * rcp_(mL - mR);

    // selection in the standard order: s_L >= 0: F_L;  else s_* >= 0: F*_L;  else s_R > 0: F*_R;  else F_R.
    // (With the acoustic p_* estimate s_L <= s_* is not guaranteed for strong compressions, so the
    //  order of the tests is part of the definition.)
    const bool left = (L.u + dsL >= T(0)) || (sst >= T(0));
    const T rK = left ? L.r : R.r;
    const T pK = left ? L.p : R.p;
    const T uK = left ? L.u : R.u;
    const T vK = left ? L.v : R.v;
    const T wK = left ? L.w : R.w;
    const T dsK = left ? dsL : dsR;
    const T mK = left ? mL : mR;
    const T sK = uK + dsK;
    const bool outer = left ? (sK >= T(0)) : !(sK > T(0));

    const T EK = pK * gc.igm1 + T(0.5) * rK * (uK * uK + vK * vK + wK * wK);
    const T inv = rcp_(sK - sst);
    const T phi = sst * inv;
    const T pstK = pK + mK * (sst - uK);
    T F0 = phi * mK;
    T F1 = pstK + F0 * sst;
    T F4 = sst * ((EK * dsK - pK * uK) * inv + pstK * (T(1) + phi));
    if (outer) {
        F0 = rK * uK;
        F1 = F0 * uK + pK;
        F4 = (EK + pK) * uK;
    }
    F[0] = F0;
    F[1] = F1;
    F[2] = F0 * vK;
    F[3] = F0 * wK;
    F[4] = F4;
}

// ---------------------------------------------------------------------------------------
// CFL rate of one cell, sum_{active d} (|v_d| + c)/dx_d  (reading S1).
template <typename T>
__device__ __forceinline__ T cfl_rate(T rho, T p, T vx, T vy, T vz, T gamma, T idx, T idy, T idz)
{
    const T c = sound_speed(gamma * p, rho);
    // inactive axes have inverse spacing 0
    return (fabs(vx) + c) * idx + (fabs(vy) + c) * idy + (fabs(vz) + c) * idz;
}

// CFL rate from a conserved state in float_t (fp32 in mixed mode: the paper computes dt
// during the variable conversion, whose output is float_t; fp64 in all-fp64 mode).
// Used by the standalone cfl kernel (T = double) and by the stage-2 epilogues.
template <typename T>
__device__ __forceinline__ T cfl_rate_from_cons(const double Un[5], const Grid& g)
{
    T r = T(Un[0]);
    r = (r < T(KH_RHO_FLOOR)) ? T(KH_RHO_FLOOR) : r;  // comparisons, not fmax: a NaN must survive
    const T ir = rcp_(r);
    const T vx = T(Un[1]) * ir, vy = T(Un[2]) * ir, vz = T(Un[3]) * ir;
    T p = T(g.gamma - 1.0) * (T(Un[4]) - T(0.5) * r * (vx * vx + vy * vy + vz * vz));
    p = (p < T(KH_P_FLOOR)) ? T(KH_P_FLOOR) : p;
    return cfl_rate<T>(r, p, vx, vy, vz, T(g.gamma), T(g.inv_dx[0]), T(g.inv_dx[1]), T(g.inv_dx[2]));
}

// ---------------------------------------------------------------------------------------
// block-wide max of a non-negative double, then one atomicMax on its bit pattern.
__device__ __forceinline__ void block_atomic_max_nonneg(double v, unsigned long long* target, double* smem32)
{
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    const int tid = threadIdx.x + blockDim.x * (threadIdx.y + blockDim.y * threadIdx.z);
    const int nthr = blockDim.x * blockDim.y * blockDim.z;
    const int lane = tid & 31, warp = tid >> 5;
    if (lane == 0) smem32[warp] = v;
    __syncthreads();
    if (warp == 0) {
        v = (lane < (nthr + 31) / 32) ? smem32[lane] : 0.0;
        for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
        if (lane == 0 && v > 0.0) atomicMax(target, (unsigned long long)__double_as_longlong(v));
    }
}

}  // namespace kh
