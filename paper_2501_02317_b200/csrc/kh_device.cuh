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

enum : int { BC_PERIODIC = 0, BC_FREE = 1, BC_OUTFLOW = 2, BC_REFLECT = 3,
             BC_COMM = 4 };   // communication boundary (Sec. 3.1.2): ghost planes supplied by the neighbouring block
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
    double p_ref;                    // reference pressure of the mixed-precision momentum flux (fp32-exact)
    int nonfinite;                   // set when a dt came out non-finite
    int pad;
};

// Number of SMs of the calling thread's current device (148 on B200): what the launch heuristics size their grids by.
// Asked once per device; falls back to the B200's 148 if the query fails.
inline int sm_count()
{
    static int cached[64] = {0};
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return 148;
    if (!cached[dev]) {
        int n = 0;
        if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) n = 148;
        cached[dev] = n;
    }
    return cached[dev];
}

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

// Explicitly rounded arithmetic: the compiler neither contracts nor re-associates these, so every
// inlined copy of the flux and slope functions computes bit-identical results from identical inputs
// (a face shared by two tiles or two slabs is evaluated by two thread blocks).
__device__ __forceinline__ float add_(float a, float b) { return __fadd_rn(a, b); }
__device__ __forceinline__ float sub_(float a, float b) { return __fadd_rn(a, -b); }
__device__ __forceinline__ float mul_(float a, float b) { return __fmul_rn(a, b); }
__device__ __forceinline__ float fma_(float a, float b, float c) { return __fmaf_rn(a, b, c); }
__device__ __forceinline__ double add_(double a, double b) { return __dadd_rn(a, b); }
__device__ __forceinline__ double sub_(double a, double b) { return __dadd_rn(a, -b); }
__device__ __forceinline__ double mul_(double a, double b) { return __dmul_rn(a, b); }
__device__ __forceinline__ double fma_(double a, double b, double c) { return __fma_rn(a, b, c); }

// c = sqrt(gamma p / rho).  fp32: gamma p * rsqrt(gamma p rho), a single MUFU.
__device__ __forceinline__ float sound_speed(float gp, float rho) { return mul_(gp, rsqrt_(mul_(gp, rho))); }
__device__ __forceinline__ double sound_speed(double gp, double rho) { return sqrt(gp / rho); }
// 1/p for the pressure ratio of Eq. 5.  fp32: t = rsqrt(gamma p rho) is the factor of the sound speed above and
// 1/p = gamma rho t^2 (multiplications instead of another MUFU; the packed kernels do the same, bit for bit).
__device__ __forceinline__ float inv_pressure(float gamma, float gp, float rho, float p)
{
    const float t = rsqrt_(mul_(gp, rho));
    return mul_(mul_(gamma, rho), mul_(t, t));
}
__device__ __forceinline__ double inv_pressure(double gamma, double gp, double rho, double p) { return 1.0 / p; }

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
// Returns the number of floor activations (0, 1 or 2).  pfl: the pressure floor (mixed precision with a reference
// pressure: mixed_pressure_floor below; otherwise the plain 1e-30).
__device__ __forceinline__ int cons_to_prim(double rho, double mx, double my, double mz, double eps,
                                            double gm1, double& p, double& vx, double& vy, double& vz,
                                            double& rho_out, double pfl = KH_P_FLOOR)
{
    int hits = 0;
    if (rho < KH_RHO_FLOOR) { rho = KH_RHO_FLOOR; hits++; }
    const double ir = 1.0 / rho;
    vx = mx * ir;
    vy = my * ir;
    vz = mz * ir;
    const double ekin = 0.5 * (mx * vx + my * vy + mz * vz);
    p = gm1 * (eps - ekin);
    if (p < pfl) { p = pfl; hits++; }
    rho_out = rho;
    return hits;
}

// Pressure floor of the one-thread-per-cell kernels (kh_simple.cuh, kh_vanleer.cuh).  Mixed precision (float_t = float,
// float2_t = double) with a reference pressure: max(1e-30, p_ref 2^-22), the floor of pr::recover (kh_pair.cuh) and of
// the tiled / TMA / strip kernels, so that floor_hits and the floored state do not depend on which kernel variant served
// the block (reading S14).  All-fp64 and all-fp32: 1e-30.
template <typename T, typename S>
__device__ __forceinline__ S mixed_pressure_floor(const Ctrl* ctrl)
{
    if constexpr (sizeof(T) == sizeof(float) && sizeof(S) == sizeof(double))
        return (S)fmax(KH_P_FLOOR, __dmul_rn(ctrl->p_ref, 0x1p-22));
    else
        return (S)KH_P_FLOOR;
}

// All-fp32 "Single" mode (float2_t = float_t = float): the same recovery on an fp32 state, every
// operation explicitly rounded (all copies of a cell return the same bits), 1/rho by MUFU.RCP.
__device__ __forceinline__ int cons_to_prim(float rho, float mx, float my, float mz, float eps, float gm1, float& p,
                                            float& vx, float& vy, float& vz, float& rho_out, float pfl = (float)KH_P_FLOOR)
{
    int hits = 0;
    if (rho < (float)KH_RHO_FLOOR) { rho = (float)KH_RHO_FLOOR; hits++; }
    const float ir = rcp_(rho);
    vx = mul_(mx, ir);
    vy = mul_(my, ir);
    vz = mul_(mz, ir);
    const float m2 = mul_(fma_(mz, mz, fma_(my, my, mul_(mx, mx))), ir);
    p = mul_(gm1, fma_(-0.5f, m2, eps));
    if (p < pfl) { p = pfl; hits++; }
    rho_out = rho;
    return hits;
}

// Eq. 3, reading S2 for ab = 0: the argument of smaller magnitude when both have
// the same sign, else 0.  fp32: FMNMX.XORSIGN gives min(|a|,|b|) carrying sign(a) xor sign(b); clamping
// at 0 keeps it only for equal signs; the sign of a is put back with one LOP3 -- three ALU instructions.
__device__ __forceinline__ float minmod(float a, float b)
{
    float t;
    asm("min.xorsign.abs.f32 %0, %1, %2;" : "=f"(t) : "f"(a), "f"(b));
    return copysignf(fmaxf(t, 0.0f), a);
}
__device__ __forceinline__ double minmod(double a, double b)
{
    const double m = fmin(fabs(a), fabs(b));
    return ((a > 0.0) == (b > 0.0) && a != 0.0 && b != 0.0) ? copysign(m, a) : 0.0;
}

// Half the limited undivided difference: (dx/2) * minmod((q0-qm)/dx, (qp-q0)/dx) on a uniform
// mesh (reading S8; PAPER.md:242 asks for Delta x in the denominator to keep the slope from
// being a difference of large products -- the undivided difference has that property too).
template <typename T>
__device__ __forceinline__ T half_slope(T qm, T q0, T qp)
{
    return mul_(T(0.5), minmod(sub_(q0, qm), sub_(qp, q0)));  // the product with 1/2 is exact
}

// Constants of the Riemann solver, computed once per kernel.
template <typename T>
struct GasConst {
    T gamma;   // gamma
    T g1;      // (gamma+1)/(2 gamma), Eq. 5
    T igm1;    // 1/(gamma-1)
    T pref;    // reference pressure: face states carry p - pref (0 in all-fp64 mode)
    __device__ __forceinline__ GasConst(double g, double p_ref)
        : gamma(T(g)), g1(T((g + 1.0) / (2.0 * g))), igm1(T(1.0 / (g - 1.0))), pref(T(p_ref)) {}
};

// Sec. 3.2.2: HLLC flux with the subtraction-safe wave speeds of Eq. 5.
//   c_K = sqrt(gamma p_K / rho_K)
//   p_* = max(0, (p_L+p_R)/2 - (u_R-u_L)/2 * rho_bar * c_bar)                        (reading S3)
//   q_K = sqrt(1 + (gamma+1)/(2 gamma) * max(p_*/p_K - 1, 0)),  Delta s_L = -c_L q_L,  Delta s_R = +c_R q_R
//   s_* = {[p_R - rho_R u_R Ds_R] - [p_L - rho_L u_L Ds_L]} / {rho_L Ds_L - rho_R Ds_R}        (Eq. 4)
// Selection in the standard order: s_L >= 0: F_L; else s_* >= 0: F*_L; else s_R > 0: F*_R; else F_R
// (with the acoustic p_* estimate s_L <= s_* is not guaranteed for strong compressions, so the order
// of the tests is part of the definition).  Flux on the selected side K, written in Ds_K throughout
// (an algebraically equivalent form of the star-state assembly, reading S4):
//   m_K = rho_K Ds_K,  p_*K = p_K + m_K (s_* - u_K),  phi = s_* / (s_K - s_*),
//   F_rho = phi m_K,  F_u = p_*K + F_rho s_*,  F_E = s_* [ (E_K Ds_K - p_K u_K)/(s_K - s_*) + p_*K (1 + phi) ],
//   F_v = F_rho v_K,  F_w = F_rho w_K;   outside the fan the upwind physical flux.
//
// Pressure enters as the deviation p' = p - pref (L.p, R.p hold p'): in the same spirit as Eq. 5, the
// momentum flux is formed without the large common term -- F_u returned here is F_u - pref, which has
// the same face-to-face differences on a uniform mesh, so that nearly uniform pressure does not cost
// the fp32 flux difference its significant digits.  With pref = 0 this is the plain form.
// F = (mass, normal momentum - pref, tangential momentum 1, tangential momentum 2, energy).
template <typename T>
__device__ __forceinline__ void hllc(const Prim<T>& L, const Prim<T>& R, const GasConst<T>& gc, T F[5])
{
    const T pL = add_(L.p, gc.pref), pR = add_(R.p, gc.pref);  // actual pressures
    const T cL = sound_speed(mul_(gc.gamma, pL), L.r);
    const T cR = sound_speed(mul_(gc.gamma, pR), R.r);

    // p_* as a deviation from pref, clipped so that the actual value is >= 0
    const T w = mul_(mul_(sub_(R.u, L.u), add_(L.r, R.r)), add_(cL, cR));
    T pst = fma_(T(-0.125), w, mul_(T(0.5), add_(L.p, R.p)));
    pst = fmax(pst, -gc.pref);

    const T qL = sqrt_(fma_(gc.g1, fmax(mul_(sub_(pst, L.p), inv_pressure(gc.gamma, mul_(gc.gamma, pL), L.r, pL)), T(0)), T(1)));
    const T qR = sqrt_(fma_(gc.g1, fmax(mul_(sub_(pst, R.p), inv_pressure(gc.gamma, mul_(gc.gamma, pR), R.r, pR)), T(0)), T(1)));
    const T dsL = -mul_(cL, qL);
    const T dsR = mul_(cR, qR);
    const T mL = mul_(L.r, dsL);
    const T mR = mul_(R.r, dsR);
    // s_* = num/den (Eq. 4) with den = m_L - m_R < 0, and 1/(s_K - s_*) = den/D with D = s_K den - num:
    // both quotients from ONE reciprocal, r = 1/(den D).  The side is chosen from signs alone.
    const T num = sub_(fma_(-mR, R.u, R.p), fma_(-mL, L.u, L.p));
    const T den = sub_(mL, mR);
    const bool left = (add_(L.u, dsL) >= T(0)) || (num <= T(0));  // s_L >= 0 or s_* >= 0
    const T rK = left ? L.r : R.r;
    const T pKd = left ? L.p : R.p;
    const T uK = left ? L.u : R.u;
    const T vK = left ? L.v : R.v;
    const T wK = left ? L.w : R.w;
    const T dsK = left ? dsL : dsR;
    const T mK = left ? mL : mR;
    const T pK = add_(pKd, gc.pref);
    const T sK = add_(uK, dsK);
    const bool outer = (left ? sK : -sK) >= T(0);  // s_L >= 0, resp. s_R <= 0

    const T D = fma_(sK, den, -num);
    const T r = rcp_(mul_(den, D));
    const T sst = mul_(num, mul_(D, r));
    const T inv = mul_(den, mul_(den, r));
    const T ke = fma_(wK, wK, fma_(vK, vK, mul_(uK, uK)));
    const T EK = fma_(pK, gc.igm1, mul_(mul_(T(0.5), rK), ke));
    const T phi = mul_(sst, inv);
    const T pstKd = fma_(mK, sub_(sst, uK), pKd);
    T F0 = mul_(phi, mK);
    T F1 = fma_(F0, sst, pstKd);
    const T A4 = fma_(EK, dsK, -mul_(pK, uK));
    T F4 = mul_(sst, fma_(A4, inv, mul_(add_(pstKd, gc.pref), add_(T(1), phi))));
    if (outer) {
        F0 = mul_(rK, uK);
        F1 = fma_(F0, uK, pKd);
        F4 = mul_(add_(EK, pK), uK);
    }
    F[0] = F0;
    F[1] = F1;
    F[2] = mul_(F0, vK);
    F[3] = mul_(F0, wK);
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
struct CflConst {
    T gm1, gamma, idx, idy, idz;
    __device__ __forceinline__ explicit CflConst(const Grid& g)
        : gm1(T(g.gamma - 1.0)), gamma(T(g.gamma)), idx(T(g.inv_dx[0])), idy(T(g.inv_dx[1])), idz(T(g.inv_dx[2])) {}
};

template <typename T, typename S = double>
__device__ __forceinline__ T cfl_rate_from_cons(const S Un[5], const CflConst<T>& cc, T* p_out = nullptr)
{
    T r = T(Un[0]);
    r = (r < T(KH_RHO_FLOOR)) ? T(KH_RHO_FLOOR) : r;  // comparisons, not fmax: a NaN must survive
    const T ir = rcp_(r);
    const T vx = T(Un[1]) * ir, vy = T(Un[2]) * ir, vz = T(Un[3]) * ir;
    T p = cc.gm1 * (T(Un[4]) - T(0.5) * r * (vx * vx + vy * vy + vz * vz));
    p = (p < T(KH_P_FLOOR)) ? T(KH_P_FLOOR) : p;
    if (p_out) *p_out = p;
    return cfl_rate<T>(r, p, vx, vy, vz, cc.gamma, cc.idx, cc.idy, cc.idz);
}

// ---------------------------------------------------------------------------------------
// Split-phase block barrier on an mbarrier in shared memory: arrive (release), do independent work,
// then wait (acquire).  All threads of the block take part in every phase.
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(count));
}
__device__ __forceinline__ unsigned long long mbar_arrive(unsigned long long* bar)
{
    unsigned long long token;
    asm volatile("mbarrier.arrive.shared::cta.b64 %0, [%1];"
                 : "=l"(token)
                 : "r"((unsigned)__cvta_generic_to_shared(bar))
                 : "memory");
    return token;
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned long long token)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t}"
        ::"r"((unsigned)__cvta_generic_to_shared(bar)), "l"(token)
        : "memory");
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
