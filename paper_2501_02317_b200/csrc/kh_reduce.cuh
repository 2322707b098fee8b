// kh_reduce.cuh -- reductions and time-step bookkeeping kernels.
#pragma once
#include "kh_device.cuh"

namespace kh {

// CFL rate maximum of the stored state, fp64 in every precision mode (S1, S7).
// Grid-stride, warp-shuffle + one atomicMax per block.  Also leaves each block's pressure sum in
// p_partial[blockIdx.x] and its pressure minimum in p_partial[gridDim.x + blockIdx.x] (fixed reduction
// order => run-to-run reproducible reference pressure).
// S = float2_t, the storage type of the state (float in the all-fp32 Single mode: converted exactly to fp64 here).
template <typename S>
__global__ void __launch_bounds__(256) cfl_rate_kernel(const S* __restrict__ U, Grid g, Ctrl* ctrl,
                                                       double* p_partial)
{
    __shared__ double red[32];
    __shared__ double psum[8], pmin[8];
    double rate = 0.0, ps = 0.0, pm = __longlong_as_double(0x7ff0000000000000LL);
    const CflConst<double> cc(g);
    for (long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x; c < g.N;
         c += (long long)gridDim.x * blockDim.x) {
        const double u[5] = {(double)U[c], (double)U[g.N + c], (double)U[2 * g.N + c], (double)U[3 * g.N + c], (double)U[4 * g.N + c]};
        double p;
        double r = cfl_rate_from_cons<double>(u, cc, &p);
        if (!(r == r)) r = __longlong_as_double(0x7ff0000000000000LL);
        rate = fmax(rate, r);
        ps += p;
        pm = fmin(pm, p);
    }
    for (int o = 16; o > 0; o >>= 1) {
        ps += __shfl_xor_sync(0xffffffffu, ps, o);
        pm = fmin(pm, __shfl_xor_sync(0xffffffffu, pm, o));
    }
    if ((threadIdx.x & 31) == 0) { psum[threadIdx.x >> 5] = ps; pmin[threadIdx.x >> 5] = pm; }
    block_atomic_max_nonneg(rate, &ctrl->rate_bits, red);  // contains a __syncthreads()
    if (threadIdx.x == 0) {
        double t = 0.0, m = pmin[0];
        for (int w = 0; w < 8; w++) { t += psum[w]; m = fmin(m, pmin[w]); }
        p_partial[blockIdx.x] = t;
        p_partial[gridDim.x + blockIdx.x] = m;
    }
}

// Reference pressure of the mixed-precision momentum flux (reading S14): min(mean pressure,
// 2 x minimum pressure), rounded to fp32 so that the fp64 primitive recovery and the fp32 Riemann solver
// use the very same number.  The stored deviation p - p_ref of a cell then has the absolute error
// ulp_fp32(|p - p_ref|) <= ulp_fp32(p) wherever p >= p_min: never worse than plain fp32 pressure, and far
// better where the pressure is nearly uniform (the mean is then below 2 p_min and is the reference).
__global__ void finish_cfl_kernel(Ctrl* ctrl, const double* p_partial, int nblocks, double inv_n)
{
    double t = 0.0, pm = p_partial[nblocks];
    for (int b = 0; b < nblocks; b++) { t += p_partial[b]; pm = fmin(pm, p_partial[nblocks + b]); }
    const float m = (float)fmin(t * inv_n, 2.0 * pm);
    ctrl->p_ref = (m == m && m > 0.0f && m < 3.0e38f) ? (double)m : 0.0;
}

// dt bookkeeping between steps of kratos_hydro_run: one thread.
//   dt = cfl / rate_max, clipped to land on t_end; t += dt; reset the reduction target.
__global__ void prepare_step_kernel(Ctrl* ctrl)
{
    const double rate = __longlong_as_double((long long)ctrl->rate_bits);
    double dt = ctrl->cfl / rate;
    if (!(dt > 0.0) || !(dt < __longlong_as_double(0x7ff0000000000000LL))) {
        ctrl->nonfinite = 1;
        dt = 0.0;
    }
    if (ctrl->t_end > 0.0) {
        const double left = ctrl->t_end - ctrl->t;
        if (left <= 0.0) dt = 0.0;
        else if (ctrl->t + dt >= ctrl->t_end) dt = left;
    }
    ctrl->dt = dt;
    if (dt > 0.0) {
        // landing exactly: t + (t_end - t) may differ from t_end in the last bit
        const double tn = ctrl->t + dt;
        ctrl->t = (ctrl->t_end > 0.0 && dt == ctrl->t_end - ctrl->t) ? ctrl->t_end : tn;
        ctrl->steps += 1;
        ctrl->rate_bits = 0ull;  // stage 2 of this step reduces the next rate
    }
}

// kratos_hydro_step(dt): the caller's dt.
__global__ void set_dt_kernel(Ctrl* ctrl, double dt)
{
    ctrl->dt = dt;
    ctrl->t += dt;
    ctrl->rate_bits = 0ull;
}

__global__ void reset_rate_kernel(Ctrl* ctrl) { ctrl->rate_bits = 0ull; }

// ---------------------------------------------------------------------------------------
// double-double accumulation (error-free transformations) for the conservation diagnostics.
struct dd {
    double hi, lo;
};
__device__ __forceinline__ dd dd_add(dd a, double b)
{
    const double s = a.hi + b;
    const double bb = s - a.hi;
    const double e = (a.hi - (s - bb)) + (b - bb);  // TwoSum
    const double lo = a.lo + e;
    const double hi = s + lo;
    return dd{hi, lo - (hi - s)};
}
__device__ __forceinline__ dd dd_add(dd a, dd b)
{
    const double s = a.hi + b.hi;
    const double bb = s - a.hi;
    const double e = (a.hi - (s - bb)) + (b.hi - bb);
    const double lo = (a.lo + b.lo) + e;
    const double hi = s + lo;
    return dd{hi, lo - (hi - s)};
}

// partial[field][block] = double-double sum of that block's share.  Launch with 256 threads.
template <typename S>
__global__ void __launch_bounds__(256) totals_kernel(const S* __restrict__ U, long long N, dd* partial)
{
    __shared__ dd red[8];
    const int field = blockIdx.y;
    const S* f = U + (long long)field * N;
    dd acc{0.0, 0.0};
    for (long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x; c < N;
         c += (long long)gridDim.x * blockDim.x)
        acc = dd_add(acc, (double)f[c]);
    for (int o = 16; o > 0; o >>= 1) {
        dd other{__shfl_xor_sync(0xffffffffu, acc.hi, o), __shfl_xor_sync(0xffffffffu, acc.lo, o)};
        acc = dd_add(acc, other);
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (lane == 0) red[warp] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        dd t = red[0];
        for (int w = 1; w < 8; w++) t = dd_add(t, red[w]);
        partial[(long long)field * gridDim.x + blockIdx.x] = t;
    }
}

// Single mode: the C-ABI carries the state as doubles; the handle stores floats.
template <typename From, typename To>
__global__ void __launch_bounds__(256) convert_state_kernel(const From* __restrict__ src, To* __restrict__ dst, long long n)
{
    for (long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x; c < n; c += (long long)gridDim.x * blockDim.x)
        dst[c] = (To)src[c];
}

// out[field] = sum over blocks, one thread per field.
__global__ void totals_final_kernel(const dd* partial, int nblocks, double* out)
{
    const int field = threadIdx.x;
    if (field >= 5) return;
    dd t{0.0, 0.0};
    for (int b = 0; b < nblocks; b++) t = dd_add(t, partial[(long long)field * nblocks + b]);
    out[field] = t.hi + t.lo;
}

}  // namespace kh
