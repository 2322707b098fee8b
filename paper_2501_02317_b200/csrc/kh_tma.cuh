// kh_tma.cuh -- KRATOS_KERNEL_TMA: the paired Heun-stage kernel (kh_pair.cuh) with every byte of global
// traffic moved by the Tensor Memory Accelerator (3D blocks, mixed precision, nx % 32 == 0, ny % 16 == 0).
//
// The arithmetic is that of kh_pair.cuh, function for function (recover, plm, hllc2: PAPER.md:163-173,
// Eq. 3, Eq. 4-5; fp64 update and Heun average: PAPER.md:232-238, 264).  What changes is how the conserved
// state gets on and off the chip.  In the paired kernel one third of the issue slots of a main warp went
// into 8-byte cp.async copies, 64-bit address arithmetic, boundary-rule branches and predicated stores.
// Here a producer warp issues, per plane of the z march,
//     one 4-D TMA box (32 x 16 x 1 x 5 doubles) for the tile,          -> raw[slot]
//     four boxes for the 2-cell halo (two row pairs, two column pairs)   -> hrow / hcol[slot]
//     one box for U0 of the plane being averaged (stage 2)               -> u0[slot]
// each completing on an mbarrier, and one TMA store per plane: the main warps write the new state over the
// raw state they just consumed (in place, same addresses, no extra buffer) and the producer ships the box.
// The main warps contain no global-memory instruction at all, the halo warps read their cells from shared
// memory, and the boundary rules of Sec. 3.1.1 become a choice of box coordinates
// (periodic wrap, clamp, mirror) made once per block plus the normal-velocity rule applied at conversion.
//
// Phases per plane k (as in kh_pair.cuh):
//                                                                            | barrier 1
//      [producer: store plane k-1, then refill its slot with plane k-1+NSLOT; halo plane k+3; U0(k+1)]
//   B) z/x/y fluxes of plane k, conversion of plane k+3, tile of plane k+1   | barrier 2
//   C) fp64 update of plane k, written in place; Heun average and CFL rate (stage 2)
//   A) of plane k+1, fused with C: x/y slopes from the primitive tile, left states published
#pragma once
#include <cuda.h>

#include <type_traits>

#include "kh_pair.cuh"

namespace kh {
namespace tma {

using pr::f2;
using pr::mk;
using pr::plm;
using pr::face_flux2;
using pr::recover;
using pr::Gas;

#ifndef KH_TMA_UNROLL
#define KH_TMA_UNROLL 4
#endif
constexpr int PTX = pr::PTX;       // 32
#ifndef KH_TMA_PTY
#define KH_TMA_PTY 16              // tile height: 16 (one block per SM) or 8 (two blocks per SM)
#endif
constexpr int PTY = KH_TMA_PTY;
constexpr int PRP = PTY / 2;       // row pairs = main warps (one or two warpgroups)
constexpr int BLOCKS_PER_SM = 16 / PTY;
static_assert(PTY == 16 || PTY == 8, "setmaxnreg acts on warpgroups: 4 or 8 main warps");
constexpr int WARP_HALO_Y = PRP;
constexpr int WARP_HALO_X = PRP + 1;
constexpr int WARP_PRODUCER = PRP + 2;
constexpr int WARP_HALO_Y2 = PRP + 3;
constexpr int NWARPS = PRP + 4;        // main warpgroup(s) + one auxiliary warpgroup (halo rows low, halo columns, producer, halo rows high):
                                       // setmaxnreg acts on whole warpgroups
constexpr int NTHREADS = NWARPS * 32;
constexpr int UNROLL = KH_TMA_UNROLL;  // planes per trip of the z march (register rotation becomes renaming)
// register split of the three warpgroups (setmaxnreg): per scheduler 2 main warps + 1 auxiliary warp <= 16384
#ifndef KH_TMA_MAIN_REGS
#define KH_TMA_MAIN_REGS 208
#endif
#ifndef KH_TMA_HALO_REGS
#define KH_TMA_HALO_REGS 72
#endif
#define KH_TMA_STR2(x) #x
#define KH_TMA_STR(x) KH_TMA_STR2(x)

template <int STAGE>
struct Cfg {
    // raw ring depth: planes k (updated in place, then stored), k+1, k+2 (held for their update), k+3 (being converted)
    // and one being refilled
    static constexpr int NSLOT = 5;
    static constexpr int NU0 = (STAGE == 2) ? 2 : 0;
    static constexpr int NHALO = (STAGE == 2 && BLOCKS_PER_SM == 2) ? 2 : 3;   // halo ring depth
};

constexpr int OWN_BYTES = 5 * PTY * PTX * 8;    // one tile box
constexpr int ROW_BYTES = 5 * 2 * PTX * 8;      // one halo row pair
constexpr int COL_BYTES = 5 * PTY * 2 * 8;      // one halo column pair

// ST = float2_t, the type the conserved state is stored in: double, or float in the all-fp32 "Single" mode (MODE 0 only).
template <int STAGE, int MODE = 0, typename ST = double>
struct Smem {
    static constexpr int NSLOT = Cfg<STAGE>::NSLOT;
    static constexpr int NHALO = Cfg<STAGE>::NHALO;
    // U0 ring: two planes for the Heun average; three for the van Leer corrector, which also stores from it (the
    // refill of a slot then never waits for the store that is still reading the previous plane)
    static constexpr int NU0 = (STAGE == 2) ? ((MODE == 2) ? 3 : 2) : 1;
    // planes in flight: fp64 conserved state, or (van Leer corrector) float_t primitives = half the bytes
    alignas(128) ST raw[NSLOT][5][(MODE == 2) ? PTY / 2 : PTY][PTX];
    alignas(128) ST u0[NU0][(STAGE == 2) ? 5 : 1][(STAGE == 2) ? PTY : 1][PTX];
    alignas(128) double hrow[NHALO][2][5][2][PTX];            // halo rows: [lo/hi][field][box row][column]
    alignas(128) double hcol[NHALO][2][5][PTY][2];            // halo columns: [lo/hi][field][row][box column]
    f2 Wt[5][PRP + 2][PTX + 4];                               // primitives of one plane, row pairs -1..PRP, columns -2..PTX+1
    f2 QLx[5][PRP][PTX + 1];                                  // left states at x faces c = 0..PTX (from column c-1)
    f2 QRxR[5][PRP];                                          // right state at x face PTX (from halo column PTX)
    float QLy[5][PRP + 1][PTX];                               // left states at y faces r = 0..PRP (from row 2r-1)
    float QRyT[5][PTX];                                       // right state at y face PRP (from halo row PTY)
    f2 Fx[5][PRP][PTX + 1];                                   // float_t fluxes through x faces (each side converts: same bits)
    float Fy[5][PRP + 1][PTX];                                // float_t fluxes through the y faces between row pairs
    double red[32];
    unsigned long long full_raw[NSLOT];
    unsigned long long full_halo[NHALO];
    unsigned long long full_u0[3];
};

// tensor maps of one stage launch (64-byte aligned kernel parameters)
struct Maps {
    CUtensorMap in_own, in_rows, in_cols;   // stage input: tile box, halo row pair, halo column pair
    CUtensorMap u0_own;                     // U0 (stage 2)
    CUtensorMap out_own;                    // stage output
    // communication boundaries in z (BC_COMM; Sec. 3.1.2): the two ghost planes of the stage input
    // beyond the low / high z face (arrays [5][2][ny][nx] the neighbouring block fills), and the neighbours' ghost
    // arrays of the stage OUTPUT (peer memory), into which this block stores its two planes next to the face
    CUtensorMap in_glo, in_ghi;
    CUtensorMap out_plo, out_phi;
};

// ---- PTX wrappers -------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait_parity(unsigned long long* bar, unsigned parity)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "W_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra D_%=;\n\t"
        "bra W_%=;\n\t"
        "D_%=:\n\t}" ::"r"(smem_u32(bar)), "r"(parity)
        : "memory");
}
__device__ __forceinline__ void tma_load4(void* dst, const CUtensorMap* map, int c0, int c1, int c2, int c3,
                                          unsigned long long* bar)
{
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];" ::
            "r"(smem_u32(dst)), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(smem_u32(bar))
        : "memory");
}
__device__ __forceinline__ void tma_store4(const CUtensorMap* map, int c0, int c1, int c2, int c3, const void* src)
{
    asm volatile("cp.async.bulk.tensor.4d.global.shared::cta.bulk_group [%0, {%1, %2, %3, %4}], [%5];" ::"l"(map),
                 "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(smem_u32(src))
                 : "memory");
}
__device__ __forceinline__ void tma_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void tma_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void tma_wait_all0() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void block_bar() { asm volatile("bar.sync 0;" ::: "memory"); }

// Stored pressure deviation of a float_t primitive (van Leer corrector): p - pref with the same two-ulp floor as
// pr::recover, so that the pressure rebuilt by the Riemann solver stays > 0.
__device__ __forceinline__ float pdev(float p, float pref_f) { return __fadd_rn(fmaxf(p, pref_f * 0x1p-22f), -pref_f); }

// Where the two halo cells beyond one side of the tile come from (Sec. 3.1.1): first source coordinate of the
// 2-wide box, the position inside the box of each of the two cells, and the normal-velocity rule.
// (Tiles start at multiples of 16 and extents are even, so the smaller source coordinate is even except for
// the clamp onto cell n-1 of the Free / Outflow rules, where both cells sit at position 1 of the box.)
struct HaloSide {
    int start, idx0, idx1, rule;
};
__device__ __forceinline__ HaloSide halo_side(int c0, int n, int bc_lo, int bc_hi, int width = 2)
{
    int r0, r1;
    const int s0 = bc_source(c0, n, bc_lo, bc_hi, r0);
    const int s1 = bc_source(c0 + 1, n, bc_lo, bc_hi, r1);
    HaloSide h;
    h.start = min(s0, s1) & ~(width - 1);  // aligned: the box stays inside the block, its first byte 16-byte aligned
                                           // (width 2 for fp64 boxes, 4 for the float boxes of the van Leer corrector)
    h.idx0 = s0 - h.start;
    h.idx1 = s1 - h.start;
    h.rule = r0;  // both cells lie beyond the same face
    return h;
}

// pr::hllc2 (Sec. 3.2.2; formulas documented at kh::hllc) for N independent face pairs in
// lock step: every statement is issued for all N before the next one, so that the N dependency chains are
// interleaved in program order and the fixed latencies of one hide behind the others.  Operation for operation
// the same arithmetic as pr::hllc2, hence the same bits.
// 1/p_K for the pressure ratio of Eq. 5.  t = rsqrt(gamma p rho) is at hand from the sound speed, and 1/p = gamma rho t^2:
// three packed multiplications instead of two more MUFU operations per face pair (the XU pipe, which also carries the
// fp32 <-> fp64 conversions, is the busiest one of this kernel).  A few ulp of error in a factor that only enters
// through max(p*/p_K - 1, 0).
#define KH_RCP_P(p, rho, t) mul2(mul2(bc(g.gamma), rho), mul2(t, t))
template <int N>
__device__ __forceinline__ void hllc2n(const f2 (&L)[N][5], const f2 (&R)[N][5], const Gas& g, f2 (&F)[N][5])
{
    using namespace pr;
    const f2 pref = bc(g.pref), one = bc(1.0f);
#define KH_EACH for (int n = 0; n < N; n++)
    f2 pL[N], pR[N], gpL[N], gpR[N], tL[N], tR[N], cL[N], cR[N], w[N], pst[N], qL[N], qR[N], dsL[N], dsR[N], mL[N], mR[N];
    f2 num[N], den[N], sL[N], rK[N], pKd[N], uK[N], vK[N], wK[N], dsK[N], mK[N], pK[N], sK[N], D[N], r[N];
    f2 sst[N], inv[N], ke[N], EK[N], phi[N], pstKd[N], F0[N], F1[N], A4[N], F4[N], G0[N], G1[N], G4[N];
    bool lx[N], ly[N], ox[N], oy[N];
#pragma unroll
    KH_EACH { pL[n] = add2(L[n][1], pref); pR[n] = add2(R[n][1], pref); }
#pragma unroll
    KH_EACH { gpL[n] = mul2(bc(g.gamma), pL[n]); gpR[n] = mul2(bc(g.gamma), pR[n]); }
#pragma unroll
    KH_EACH { tL[n] = rsqrt2(mul2(gpL[n], L[n][0])); tR[n] = rsqrt2(mul2(gpR[n], R[n][0])); }
#pragma unroll
    KH_EACH { cL[n] = mul2(gpL[n], tL[n]); cR[n] = mul2(gpR[n], tR[n]); }
#pragma unroll
    KH_EACH w[n] = mul2(mul2(sub2(R[n][2], L[n][2]), add2(L[n][0], R[n][0])), add2(cL[n], cR[n]));
#pragma unroll
    KH_EACH pst[n] = maxs(fma2(bc(-0.125f), w[n], mul2(bc(0.5f), add2(L[n][1], R[n][1]))), -g.pref);
#pragma unroll
    KH_EACH {
        qL[n] = sqrt2(fma2(bc(g.g1), max0(mul2(sub2(pst[n], L[n][1]), KH_RCP_P(pL[n], L[n][0], tL[n]))), one));
        qR[n] = sqrt2(fma2(bc(g.g1), max0(mul2(sub2(pst[n], R[n][1]), KH_RCP_P(pR[n], R[n][0], tR[n]))), one));
    }
#pragma unroll
    KH_EACH { dsL[n] = neg2(mul2(cL[n], qL[n])); dsR[n] = mul2(cR[n], qR[n]); }
#pragma unroll
    KH_EACH { mL[n] = mul2(L[n][0], dsL[n]); mR[n] = mul2(R[n][0], dsR[n]); }
#pragma unroll
    KH_EACH {
        num[n] = sub2(fma2(neg2(mR[n]), R[n][2], R[n][1]), fma2(neg2(mL[n]), L[n][2], L[n][1]));
        den[n] = sub2(mL[n], mR[n]);
        sL[n] = add2(L[n][2], dsL[n]);
    }
#pragma unroll
    KH_EACH {
        lx[n] = (sL[n].x >= 0.0f) || (num[n].x <= 0.0f);
        ly[n] = (sL[n].y >= 0.0f) || (num[n].y <= 0.0f);
    }
#pragma unroll
    KH_EACH {
        rK[n] = sel(lx[n], ly[n], L[n][0], R[n][0]); pKd[n] = sel(lx[n], ly[n], L[n][1], R[n][1]);
        uK[n] = sel(lx[n], ly[n], L[n][2], R[n][2]); vK[n] = sel(lx[n], ly[n], L[n][3], R[n][3]);
        wK[n] = sel(lx[n], ly[n], L[n][4], R[n][4]); dsK[n] = sel(lx[n], ly[n], dsL[n], dsR[n]);
        mK[n] = sel(lx[n], ly[n], mL[n], mR[n]);
    }
#pragma unroll
    KH_EACH { pK[n] = add2(pKd[n], pref); sK[n] = add2(uK[n], dsK[n]); }
#pragma unroll
    KH_EACH {
        ox[n] = (lx[n] ? sK[n].x : -sK[n].x) >= 0.0f;
        oy[n] = (ly[n] ? sK[n].y : -sK[n].y) >= 0.0f;
        D[n] = fma2(sK[n], den[n], neg2(num[n]));
    }
#pragma unroll
    KH_EACH r[n] = rcp2(mul2(den[n], D[n]));
#pragma unroll
    KH_EACH { sst[n] = mul2(num[n], mul2(D[n], r[n])); inv[n] = mul2(den[n], mul2(den[n], r[n])); }
#pragma unroll
    KH_EACH {
        ke[n] = fma2(wK[n], wK[n], fma2(vK[n], vK[n], mul2(uK[n], uK[n])));
        EK[n] = fma2(pK[n], bc(g.igm1), mul2(mul2(bc(0.5f), rK[n]), ke[n]));
    }
#pragma unroll
    KH_EACH { phi[n] = mul2(sst[n], inv[n]); pstKd[n] = fma2(mK[n], sub2(sst[n], uK[n]), pKd[n]); }
#pragma unroll
    KH_EACH { F0[n] = mul2(phi[n], mK[n]); A4[n] = fma2(EK[n], dsK[n], neg2(mul2(pK[n], uK[n]))); }
#pragma unroll
    KH_EACH {
        F1[n] = fma2(F0[n], sst[n], pstKd[n]);
        F4[n] = mul2(sst[n], fma2(A4[n], inv[n], mul2(add2(pstKd[n], pref), add2(one, phi[n]))));
    }
#pragma unroll
    KH_EACH { G0[n] = mul2(rK[n], uK[n]); G4[n] = mul2(add2(EK[n], pK[n]), uK[n]); }
#pragma unroll
    KH_EACH G1[n] = fma2(G0[n], uK[n], pKd[n]);
#pragma unroll
    KH_EACH {
        F0[n] = sel(ox[n], oy[n], G0[n], F0[n]);
        F1[n] = sel(ox[n], oy[n], G1[n], F1[n]);
        F4[n] = sel(ox[n], oy[n], G4[n], F4[n]);
    }
#pragma unroll
    KH_EACH {
        F[n][0] = F0[n]; F[n][1] = F1[n]; F[n][2] = mul2(F0[n], vK[n]); F[n][3] = mul2(F0[n], wK[n]); F[n][4] = F4[n];
    }
#undef KH_EACH
}

// states in the global frame (rho, p - pref, vx, vy, vz) -> face-normal frame of axis DIR, and the flux back
template <int DIR>
__device__ __forceinline__ void to_normal(const f2 q[5], f2 o[5])
{
    constexpr int iu = 2 + DIR, iv = 2 + (DIR + 1) % 3, iw = 2 + (DIR + 2) % 3;
    o[0] = q[0]; o[1] = q[1]; o[2] = q[iu]; o[3] = q[iv]; o[4] = q[iw];
}
template <int DIR>
__device__ __forceinline__ void from_normal(const f2 F[5], f2 Fo[5])
{
    constexpr int iu = 2 + DIR, iv = 2 + (DIR + 1) % 3, iw = 2 + (DIR + 2) % 3;
    Fo[0] = F[0]; Fo[iu - 1] = F[1]; Fo[iv - 1] = F[2]; Fo[iw - 1] = F[3]; Fo[4] = F[4];
}

// One Heun stage.  STAGE 1: Uout = Uin + dt L(Uin).  STAGE 2: Uout = 1/2 U0 + 1/2 (Uin + dt L(Uin))
// (Uout aliases U0) and the CFL rate maximum of Uout.  3D only.
// Face states of a cell: Eq. 3 slopes (MODE 0) or piecewise-constant states (MODE 1, van Leer predictor).
template <int MODE>
__device__ __forceinline__ void plm_m(f2 qm, f2 q, f2 qp, f2& qL, f2& qR)
{
    if (MODE == 1) { qL = q; qR = q; }
    else plm(qm, q, qp, qL, qR);
}

// MODE 0: Heun stage.  MODE 1 (with STAGE 1): predictor of the van Leer integrator (Sec. 3.3, reading
// S15): piecewise-constant face states (all slopes zero), half a time step, and the result leaves as float_t
// primitives W^{n+1/2} = prim(U + dt/2 L_1(U)) (a float box written over the consumed raw plane and stored by TMA).
// MODE 2 (with STAGE 2): its corrector U^{n+1} = U^n + dt L_2(W^{n+1/2}): the plane ring and the halo boxes carry the
// float_t primitives (no recovery, no fp64 chain), U^n arrives through the U0 ring, is updated in place there and stored.
// COMM: the block has communication boundaries in z (a separate instantiation: the undivided block pays nothing for them).
template <int STAGE, int MODE = 0, typename ST = double, bool COMM = false>
__global__ void __launch_bounds__(NTHREADS, BLOCKS_PER_SM)
stage_tma(const __grid_constant__ Maps maps, Grid g, Ctrl* ctrl, int zchunk)
{
    static_assert(MODE == 0 || (MODE == 1 && STAGE == 1) || (MODE == 2 && STAGE == 2),
                  "the van Leer predictor has the data flow of stage 1, the corrector that of stage 2");
    constexpr bool SGL = sizeof(ST) == 4;          // all-fp32 "Single" mode: fp32 state, update and boxes
    static_assert(!SGL || MODE == 0, "the fp32 state comes with the Heun integrator only");
    constexpr bool FBOX = SGL || MODE == 2;        // the stage input arrives as float boxes
    using S = Smem<STAGE, MODE, ST>;
    using ST2 = typename std::conditional<SGL, float2, double2>::type;
    constexpr int NU0 = S::NU0;
    constexpr int NSLOT = S::NSLOT;
    constexpr int NHALO = S::NHALO;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    S& sm = *reinterpret_cast<S*>(smem_raw);

    const double dt = (MODE == 1) ? 0.5 * ctrl->dt : ctrl->dt;
    if (!(dt > 0.0)) return;  // a step clipped to zero length (run_until past t_end) does nothing
    const double pref_d = SGL ? 0.0 : ctrl->p_ref;   // (fp32 state: the deviation from a reference pressure gains nothing)
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int nx = g.n[0], ny = g.n[1], nz = g.n[2];
    const int i0 = blockIdx.x * PTX, j0 = blockIdx.y * PTY;
    const int kbeg = blockIdx.z * zchunk;
    const int kend = min(kbeg + zchunk, nz);
    const int kfirst = kbeg - 1;  // priming iteration: builds the tile of plane kbeg
    const int pbase = kbeg - 2;   // first plane of the raw ring: plane p sits in slot (p - pbase) % NSLOT
    const ST gm1 = ST(g.gamma - 1.0);
    const ST pref_s = ST(pref_d);
    Gas gas;
    gas.gamma = (float)g.gamma;
    gas.g1 = (float)((g.gamma + 1.0) / (2.0 * g.gamma));
    gas.igm1 = (float)(1.0 / (g.gamma - 1.0));
    gas.pref = (float)pref_d;

    if (threadIdx.x == 0) {
        for (int s = 0; s < NSLOT; s++) mbar_init(&sm.full_raw[s], 1);
        for (int s = 0; s < NHALO; s++) mbar_init(&sm.full_halo[s], 1);
        for (int s = 0; s < 3; s++) mbar_init(&sm.full_u0[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    int hits = 0;
    f2 rate = mk(0.0f, 0.0f);

    if (warp < PRP) {
        // ================================ main warps: cells (i, ja), (i, ja+1) ========================
        asm volatile("setmaxnreg.inc.sync.aligned.u32 " KH_TMA_STR(KH_TMA_MAIN_REGS) ";");
        const int w = warp;
        constexpr int RAWF = PTY * PTX, RAWS = 5 * RAWF;              // element strides of raw / u0: field, slot
        constexpr int WTF = (PRP + 2) * (PTX + 4);                    // f2 field stride of Wt
        constexpr int QXF = PRP * (PTX + 1);                          // f2 field stride of QLx, double2 of Fx
        constexpr int QYF = (PRP + 1) * PTX;                          // field stride of QLy (float) and Fy (double)
        ST* const raw0 = (MODE == 2) ? &sm.raw[0][0][0][0]            // (float planes: addressed in convert)
                                     : &sm.raw[0][0][2 * w][lane];     // row 2w; row 2w+1 is + PTX
        const ST* const u00 = &sm.u0[0][0][(STAGE == 2) ? 2 * w : 0][lane];
        f2* const wt = &sm.Wt[0][w + 1][lane + 2];
        f2* const qlx = &sm.QLx[0][w][lane];      // left state of the own low x face; own high face is + 1
        float* const qly = &sm.QLy[0][w][lane];   // left state of the pair's low y face; the pair's high face is + PTX
        f2* const fxs = &sm.Fx[0][w][lane];
        float* const fys = &sm.Fy[0][w][lane];

        const ST dtdx = ST(dt * g.inv_dx[0]), dtdy = ST(dt * g.inv_dx[1]), dtdz = ST(dt * g.inv_dx[2]);
        const CflConst<float> cc(g);

        // conversion of plane kk (ring index q = kk - pbase): wait for its box, recover the pair's primitives
        auto convert = [&](int kk, int slot, unsigned parity, f2 W[5], bool count) {
            int rz = VN_KEEP;
            if (kk < 0 || kk >= nz) (void)bc_source(kk, nz, g.bc[4], g.bc[5], rz);
            mbar_wait_parity(&sm.full_raw[slot], parity);
            if (MODE == 2) {  // the ring slot holds a float box [5][PTY][PTX] of primitives (rho, p, vx, vy, vz)
                const float* sf = reinterpret_cast<const float*>(&sm.raw[0][0][0][0]) + slot * RAWS + (2 * w * PTX + lane);
                const float pref_f = (float)pref_d;
#pragma unroll
                for (int f = 0; f < 5; f++) W[f] = mk(sf[f * RAWF], sf[f * RAWF + PTX]);
                W[1] = mk(pdev(W[1].x, pref_f), pdev(W[1].y, pref_f));
                W[4] = mk(apply_vn_rule(W[4].x, rz), apply_vn_rule(W[4].y, rz));
                return;
            }
            const ST* s = raw0 + slot * RAWS;
            ST ua[5], ub[5];
#pragma unroll
            for (int f = 0; f < 5; f++) { ua[f] = s[f * RAWF]; ub[f] = s[f * RAWF + PTX]; }
            float Wa[5], Wb[5];
            const int ha = recover(ua[0], ua[1], ua[2], ua[3], ua[4], gm1, pref_s, VN_KEEP, VN_KEEP, rz, Wa);
            const int hb = recover(ub[0], ub[1], ub[2], ub[3], ub[4], gm1, pref_s, VN_KEEP, VN_KEEP, rz, Wb);
            if (count) hits += ha + hb;
#pragma unroll
            for (int f = 0; f < 5; f++) W[f] = mk(Wa[f], Wb[f]);
        };

        // ---- prologue: planes kbeg-2 .. kbeg+1 (ring slots 0 .. 3, first fill: parity 0) ----
        f2 Wa[5], Wb[5], Wn[5], QLz[5];   // W(k), W(k+1), W(k+2), left state of z face k+1/2
        ST2 Fzlo[5];               // dt/dz * flux through z face k-1/2
        {
            f2 Wm[5];
            convert(kbeg - 2, 0, 0u, Wm, false);
            convert(kbeg - 1, 1, 0u, Wa, false);
            convert(kbeg, 2, 0u, Wb, true);
            convert(kbeg + 1, 3, 0u, Wn, kbeg + 1 < kend);
#pragma unroll
            for (int f = 0; f < 5; f++) {
                f2 qR;
                plm_m<MODE>(Wm[f], Wa[f], Wb[f], QLz[f], qR);
                Fzlo[f].x = Fzlo[f].y = ST(0);
            }
        }
        // ring positions of the planes k+3 (converted) and k (updated) at the first iteration k = kfirst
        constexpr int QCONV = 4;   // ring index of the plane converted in the first iteration (kbeg+2)
        int s_conv = QCONV % NSLOT, s_upd = 1;
        unsigned par_conv = (QCONV >= NSLOT) ? 1u : 0u;

        f2 QRx[5], QRy[5];
        float QLyo[5];  // left state of the face between the pair's two cells
        ST2 dU[5];
#pragma unroll
        for (int f = 0; f < 5; f++) { QRx[f] = QRy[f] = mk(0.f, 0.f); QLyo[f] = 0.f; dU[f].x = dU[f].y = ST(0); }

#pragma unroll UNROLL
        for (int k = kfirst; k < kend; k++) {
            const bool live = k >= kbeg;
            block_bar();
            // ---------------- phase B: fluxes of plane k, tile of plane k+1 ----------------
            // The z, x and y Riemann problems of the pair are independent: they are solved in lock step
            // (hllc2n).  In the priming iteration the x / y inputs are not valid yet; those results are
            // computed all the same (one basic block) and never used.
            ST2 Fzhi[5];
            f2 Wn2[5];
            {
                f2 L[3][5], R[3][5], Fn[3][5], F[5];
                {
                    f2 qL[5], qR[5];
#pragma unroll
                    for (int f = 0; f < 5; f++) {
                        qL[f] = QLz[f];
                        plm_m<MODE>(Wa[f], Wb[f], Wn[f], QLz[f], qR[f]);
                    }
                    to_normal<2>(qL, L[0]);
                    to_normal<2>(qR, R[0]);
#pragma unroll
                    for (int f = 0; f < 5; f++) qL[f] = qlx[f * QXF];
                    to_normal<0>(qL, L[1]);
                    to_normal<0>(QRx, R[1]);
#pragma unroll
                    for (int f = 0; f < 5; f++) qL[f] = mk(qly[f * QYF], QLyo[f]);
                    to_normal<1>(qL, L[2]);
                    to_normal<1>(QRy, R[2]);
                }
                hllc2n<3>(L, R, gas, Fn);
                // plane k+3 (Sec. 3.1): converted here, where the registers of the Riemann solver are free again; its
                // fp64 chain overlaps the flux accumulation below and phase B(k+1) starts with W(k+3) at hand
                convert(k + 3, s_conv, par_conv, Wn2, k + 3 < kend);
                from_normal<2>(Fn[0], F);
#pragma unroll
                for (int f = 0; f < 5; f++) {
                    Fzhi[f].x = mul_(dtdz, (ST)F[f].x); Fzhi[f].y = mul_(dtdz, (ST)F[f].y);
                    dU[f].x = sub_(Fzlo[f].x, Fzhi[f].x); dU[f].y = sub_(Fzlo[f].y, Fzhi[f].y);
                }
                from_normal<0>(Fn[1], F);
#pragma unroll
                for (int f = 0; f < 5; f++) {
                    fxs[f * QXF] = F[f];
                    dU[f].x = fma_(dtdx, (ST)F[f].x, dU[f].x);
                    dU[f].y = fma_(dtdx, (ST)F[f].y, dU[f].y);
                }
                from_normal<1>(Fn[2], F);
#pragma unroll
                for (int f = 0; f < 5; f++) {
                    const ST flo = (ST)F[f].x, fin = (ST)F[f].y;
                    fys[f * QYF] = F[f].x;
                    dU[f].x = fma_(dtdy, sub_(flo, fin), dU[f].x);
                    dU[f].y = fma_(dtdy, fin, dU[f].y);
                }
            }
            if (k + 1 < kend) {
#pragma unroll
                for (int f = 0; f < 5; f++) wt[f * WTF] = Wb[f];
            }
            // The thread's own fp64 data for the update (nobody else touches these entries) are fetched BEFORE the barrier:
            // their latency hides behind the barrier wait and they stay out of the load burst that follows it.
            ST* const su = raw0 + s_upd * RAWS;
            const int m0 = max(k - kbeg, 0);
            const ST* const s0 = u00 + (m0 % NU0) * RAWS;
            if (STAGE == 2 && live) mbar_wait_parity(&sm.full_u0[m0 % NU0], (unsigned)(m0 / NU0) & 1u);
            ST ua[5], ub[5], va[5], vb[5];
#pragma unroll
            for (int f = 0; f < 5; f++) {
                if (MODE != 2) {
                    ua[f] = su[f * RAWF];
                    ub[f] = su[f * RAWF + PTX];
                }
                if (STAGE == 2) { va[f] = s0[f * RAWF]; vb[f] = s0[f * RAWF + PTX]; }
            }
            block_bar();
            // ---------------- phase C of plane k + phase A of plane k+1, as one block of straight-line code ----------
            // C: fp64 update of plane k, written in place, explicitly rounded so that the result
            //    does not depend on what the compiler contracts.
            // A: x / y slopes of plane k+1 from the tile written in phase B, left states published for phase B(k+1).
            // The two are independent; all shared-memory loads come first and all stores last (the compiler cannot
            // reorder them itself), so that their latencies overlap.  In the priming iteration C works on stale
            // data and in the last iteration A does: both results are never used (the in-place write then lands in
            // a slot whose plane has been converted already and is refilled later).
            {
                f2 fxh[5];
                float fyh[5];
                f2 xm[5], xp[5], qLx[5], qLy[5];
                float below[5], above[5];   // rows 2w-1 and 2w+2: the near halves of the neighbouring row pairs
#pragma unroll
                for (int f = 0; f < 5; f++) {
                    fxh[f] = fxs[f * QXF + 1];
                    fyh[f] = fys[f * QYF + PTX];
                }
#pragma unroll
                for (int f = 0; f < 5; f++) {
                    xm[f] = wt[f * WTF - 1];
                    xp[f] = wt[f * WTF + 1];
                    below[f] = wt[f * WTF - (PTX + 4)].y;
                    above[f] = wt[f * WTF + (PTX + 4)].x;
                }
#pragma unroll
                for (int f = 0; f < 5; f++) {
                    // the state the flux differences are added to: the stage input (Heun), U^n (van Leer corrector)
                    const ST ba = (MODE == 2) ? va[f] : ua[f], bb = (MODE == 2) ? vb[f] : ub[f];
                    ST xa = add_(ba, fma_(-dtdx, (ST)fxh[f].x, dU[f].x));
                    ST xb = add_(bb, fma_(-dtdy, (ST)fyh[f], fma_(-dtdx, (ST)fxh[f].y, dU[f].y)));
                    if (STAGE == 2 && MODE == 0) {
                        xa = fma_(ST(0.5), va[f], mul_(ST(0.5), xa));
                        xb = fma_(ST(0.5), vb[f], mul_(ST(0.5), xb));
                    }
                    ua[f] = xa;
                    ub[f] = xb;
                }
                if (STAGE == 2) {  // CFL rate of the new state (readings S1/S7), both cells at once; no branch:
                                   // the priming iteration computes it on stale data and drops it
                    using namespace pr;
                    const float rfl = (float)KH_RHO_FLOOR, pfl = (float)KH_P_FLOOR;
                    f2 r = mk((float)ua[0], (float)ub[0]);
                    r = mk(r.x < rfl ? rfl : r.x, r.y < rfl ? rfl : r.y);  // comparisons, not fmax: a NaN must survive
                    const f2 ir = rcp2(r);
                    const f2 vx = mul2(mk((float)ua[1], (float)ub[1]), ir);
                    const f2 vy = mul2(mk((float)ua[2], (float)ub[2]), ir);
                    const f2 vz = mul2(mk((float)ua[3], (float)ub[3]), ir);
                    const f2 v2 = fma2(vz, vz, fma2(vy, vy, mul2(vx, vx)));
                    f2 p = mul2(bc(cc.gm1), fma2(mul2(bc(-0.5f), r), v2, mk((float)ua[4], (float)ub[4])));
                    p = mk(p.x < pfl ? pfl : p.x, p.y < pfl ? pfl : p.y);
                    const f2 gp = mul2(bc(cc.gamma), p);
                    const f2 c = mul2(gp, rsqrt2(mul2(gp, r)));
                    const f2 ax = mk(fabsf(vx.x), fabsf(vx.y)), ay = mk(fabsf(vy.x), fabsf(vy.y)),
                             az = mk(fabsf(vz.x), fabsf(vz.y));
                    f2 rt = mul2(add2(ax, c), bc(cc.idx));
                    rt = fma2(add2(ay, c), bc(cc.idy), rt);
                    rt = fma2(add2(az, c), bc(cc.idz), rt);
                    if (!(rt.x == rt.x)) rt.x = __int_as_float(0x7f800000);
                    if (!(rt.y == rt.y)) rt.y = __int_as_float(0x7f800000);
                    rate = mk(live ? fmaxf(rate.x, rt.x) : rate.x, live ? fmaxf(rate.y, rt.y) : rate.y);
                }
#pragma unroll
                for (int f = 0; f < 5; f++) {
                    const f2 q = Wb[f];  // W(k+1)
                    plm_m<MODE>(xm[f], q, xp[f], qLx[f], QRx[f]);
                    if (MODE == 1) { qLy[f] = q; QRy[f] = q; }
                    else pr::plm_along_pair(below[f], q, above[f], qLy[f], QRy[f]);
                    QLyo[f] = qLy[f].x;
                }
                if (MODE == 1) {
                    // W^{n+1/2} as float_t primitives (actual pressure: offset 0), written as a float box [5][PTY][PTX]
                    // over the head of the raw plane just consumed (every thread read its entries before barrier 2)
                    float Wpa[5], Wpb[5];
                    const int ha = recover(ua[0], ua[1], ua[2], ua[3], ua[4], gm1, ST(0), VN_KEEP, VN_KEEP, VN_KEEP, Wpa);
                    const int hb = recover(ub[0], ub[1], ub[2], ub[3], ub[4], gm1, ST(0), VN_KEEP, VN_KEEP, VN_KEEP, Wpb);
                    if (live) hits += ha + hb;
                    float* const sf = reinterpret_cast<float*>(raw0 + s_upd * RAWS - (2 * w * PTX + lane)) + (2 * w * PTX + lane);
#pragma unroll
                    for (int f = 0; f < 5; f++) {
                        sf[f * RAWF] = Wpa[f];
                        sf[f * RAWF + PTX] = Wpb[f];
                    }
                }
#pragma unroll
                for (int f = 0; f < 5; f++) {
                    if (MODE == 0) {
                        su[f * RAWF] = ua[f];
                        su[f * RAWF + PTX] = ub[f];
                    }
                    if (MODE == 2 && live) {  // U^{n+1} over U^n in the U0 ring: the producer ships that box
                        ST* const sv = const_cast<ST*>(s0);
                        sv[f * RAWF] = ua[f];
                        sv[f * RAWF + PTX] = ub[f];
                    }
                    qlx[f * QXF + 1] = qLx[f];
                    qly[f * QYF + PTX] = qLy[f].y;
                }
                fence_async_smem();  // the producer ships the updated box after the next barrier
            }
            // rotate the z march and the ring
#pragma unroll
            for (int f = 0; f < 5; f++) {
                Wa[f] = Wb[f]; Wb[f] = Wn[f]; Fzlo[f] = Fzhi[f];
                Wn[f] = Wn2[f];
            }
            if (++s_conv == NSLOT) { s_conv = 0; par_conv ^= 1u; }
            if (++s_upd == NSLOT) s_upd = 0;
        }
        block_bar();  // the producer ships the last plane after this barrier
    } else {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 " KH_TMA_STR(KH_TMA_HALO_REGS) ";");
    if (warp == WARP_HALO_Y || warp == WARP_HALO_Y2) {
        // ============ halo rows: warp HALO_Y owns rows -2, -1, warp HALO_Y2 rows PTY, PTY+1 (lane = column) ============
        const bool top = (warp == WARP_HALO_Y2);
        const HaloSide hsd = top ? halo_side(j0 + PTY, ny, g.bc[2], g.bc[3]) : halo_side(j0 - 2, ny, g.bc[2], g.bc[3]);
        constexpr int HF = 2 * PTX, HSIDE = 5 * HF, HSLOT = 2 * HSIDE;   // double strides of hrow: field, side, slot
        const int off0 = (top ? HSIDE : 0) + hsd.idx0 * PTX + lane, off1 = (top ? HSIDE : 0) + hsd.idx1 * PTX + lane;
        const int ry = hsd.rule;
        const double* const h0 = &sm.hrow[0][0][0][0][0];
        constexpr int WTF = (PRP + 2) * (PTX + 4);
        constexpr int QYF = (PRP + 1) * PTX;
        f2* const wown = &sm.Wt[0][top ? PRP + 1 : 0][lane + 2];                 // the warp's own row pair of the tile
        const f2* const wnext = wown + (top ? -(PTX + 4) : (PTX + 4));          // the tile's row pair next to it
        float W0[5], W1[5];   // the two rows, low row first
#pragma unroll
        for (int f = 0; f < 5; f++) W0[f] = W1[f] = 0.0f;
        int hs = 0;
        unsigned hpar = 0u;
#pragma unroll 1
        for (int k = kfirst; k < kend; k++) {
            const bool live = k >= kbeg;
            // phase A: limited y state of the row next to the tile (row -1 resp. PTY) of plane k
            if (live) {
                f2 nb[5];
#pragma unroll
                for (int f = 0; f < 5; f++) nb[f] = wnext[f * WTF];
#pragma unroll
                for (int f = 0; f < 5; f++) {
                    // bottom: rows (-2, -1, 0) -> left state of the tile's low y face; top: rows (PTY-1, PTY, PTY+1)
                    // -> right state of the tile's high y face
                    const float qm = top ? nb[f].y : W0[f], q = top ? W0[f] : W1[f], qp = top ? W1[f] : nb[f].x;
                    f2 qL, qR;
                    plm_m<MODE>(mk(qm, qm), mk(q, q), mk(qp, qp), qL, qR);
                    if (top) sm.QRyT[f][lane] = qR.x;
                    else     sm.QLy[f][0][lane] = qL.x;
                }
            }
            block_bar();
            // phase B: (top) flux through the tile's high y face of plane k; halo rows of plane k+1
            if (live && top) {
                // One packed Riemann call for both high edges of the tile: component .x solves the y face above
                // column `lane` (32 faces), component .y of lanes 0..PTY-1 the x face right of row `lane`.
                const int xr = min(lane, PTY - 1);
                const float* const qlx_e = reinterpret_cast<const float*>(&sm.QLx[0][xr >> 1][PTX]) + (xr & 1);
                const float* const qrx_e = reinterpret_cast<const float*>(&sm.QRxR[0][xr >> 1]) + (xr & 1);
                constexpr int QXF2 = 2 * PRP * (PTX + 1), QRF2 = 2 * PRP;   // float strides of QLx / QRxR per field
                float yl[5], yr[5], xl[5], xrr[5];
#pragma unroll
                for (int f = 0; f < 5; f++) {
                    yl[f] = sm.QLy[f][PRP][lane];
                    yr[f] = sm.QRyT[f][lane];
                    xl[f] = qlx_e[f * QXF2];
                    xrr[f] = qrx_e[f * QRF2];
                }
                // face-normal frames: y face (rho, p, vy, vz, vx), x face (rho, p, vx, vy, vz)
                const f2 L[5] = {mk(yl[0], xl[0]), mk(yl[1], xl[1]), mk(yl[3], xl[2]), mk(yl[4], xl[3]), mk(yl[2], xl[4])};
                const f2 R[5] = {mk(yr[0], xrr[0]), mk(yr[1], xrr[1]), mk(yr[3], xrr[2]), mk(yr[4], xrr[3]), mk(yr[2], xrr[4])};
                f2 F[5];
                pr::hllc2(L, R, gas, F);
                // back to conserved-field order: y face (F0, F4', F1, F3', F4) with normal momentum in slot 2
                sm.Fy[0][PRP][lane] = F[0].x;
                sm.Fy[2][PRP][lane] = F[1].x;
                sm.Fy[3][PRP][lane] = F[2].x;
                sm.Fy[1][PRP][lane] = F[3].x;
                sm.Fy[4][PRP][lane] = F[4].x;
                if (lane < PTY) {
                    float* const fxe = reinterpret_cast<float*>(&sm.Fx[0][lane >> 1][PTX]) + (lane & 1);
                    constexpr int FXF2 = 2 * PRP * (PTX + 1);   // float stride of Fx per field
#pragma unroll
                    for (int f = 0; f < 5; f++) fxe[f * FXF2] = F[f].y;
                }
            }
            if (k + 1 < kend) {
                mbar_wait_parity(&sm.full_halo[hs], hpar);
                const double* s = h0 + hs * HSLOT;
                if (FBOX) {  // float boxes: [side][field][box row][column], 1280 bytes per side
                    const float* sf = reinterpret_cast<const float*>(s) + (top ? 5 * 2 * PTX : 0) + lane;
                    const float pref_f = (float)pref_d;
#pragma unroll
                    for (int f = 0; f < 5; f++) { W0[f] = sf[f * 2 * PTX + hsd.idx0 * PTX]; W1[f] = sf[f * 2 * PTX + hsd.idx1 * PTX]; }
                    if (SGL) {  // conserved fp32 state
                        float c0[5], c1[5];
#pragma unroll
                        for (int f = 0; f < 5; f++) { c0[f] = W0[f]; c1[f] = W1[f]; }
                        (void)recover(c0[0], c0[1], c0[2], c0[3], c0[4], (float)gm1, pref_f, VN_KEEP, ry, VN_KEEP, W0);
                        (void)recover(c1[0], c1[1], c1[2], c1[3], c1[4], (float)gm1, pref_f, VN_KEEP, ry, VN_KEEP, W1);
                    } else {    // float_t primitives of the van Leer predictor
                        W0[1] = pdev(W0[1], pref_f); W1[1] = pdev(W1[1], pref_f);
                        W0[3] = apply_vn_rule(W0[3], ry);  W1[3] = apply_vn_rule(W1[3], ry);
                    }
                } else {
                double u0[5], u1[5];
#pragma unroll
                for (int f = 0; f < 5; f++) { u0[f] = s[off0 + f * HF]; u1[f] = s[off1 + f * HF]; }
                (void)recover(u0[0], u0[1], u0[2], u0[3], u0[4], (double)gm1, pref_d, VN_KEEP, ry, VN_KEEP, W0);
                (void)recover(u1[0], u1[1], u1[2], u1[3], u1[4], (double)gm1, pref_d, VN_KEEP, ry, VN_KEEP, W1);
                }
#pragma unroll
                for (int f = 0; f < 5; f++) wown[f * WTF] = mk(W0[f], W1[f]);
                if (++hs == NHALO) { hs = 0; hpar ^= 1u; }
            }
            block_bar();
        }
        block_bar();
    } else if (warp == WARP_HALO_X) {
        // ================================ halo columns -2, -1, PTX, PTX+1 =============================
        const int cid = lane & 3, rp = min(lane >> 2, PRP - 1);     // column id, row pair
        const bool xact = (lane >> 2) < PRP;                        // (a tile of 8 rows keeps half the lanes busy)
        const int col = (cid < 2) ? cid - 2 : PTX + cid - 2;
        constexpr int XW = FBOX ? 4 : 2;   // width of the halo column boxes (16 bytes: 2 doubles or 4 floats)
        const HaloSide side = (cid < 2) ? halo_side(i0 - 2, nx, g.bc[0], g.bc[1], XW) : halo_side(i0 + PTX, nx, g.bc[0], g.bc[1], XW);
        const int bidx = (cid & 1) ? side.idx1 : side.idx0;
        const int rx = side.rule;
        constexpr int CF = PTY * 2, CSIDE = 5 * CF, CSLOT = 2 * CSIDE;   // double strides of hcol: field, side, slot
        const double* const c0 = &sm.hcol[0][0][0][0][0] + (cid >> 1) * CSIDE + (2 * rp) * 2 + bidx;
        constexpr int WTF = (PRP + 2) * (PTX + 4);
        f2* const wt = &sm.Wt[0][rp + 1][col + 2];
        const int dl = (cid == 0) ? 0 : -1, dr = (cid == 3) ? 0 : 1;   // neighbours inside the tile array
        f2 W[5];
#pragma unroll
        for (int f = 0; f < 5; f++) W[f] = mk(0.f, 0.f);
        int hs = 0;
        unsigned hpar = 0u;
#pragma unroll 1
        for (int k = kfirst; k < kend; k++) {
            const bool live = k >= kbeg;
            // phase A: limited x states of columns -1 and PTX of plane k
            if (live) {
                // loads first, stores last: the shared-memory pipe is busiest in this window and every load this warp
                // waits for on its own is time the main warps spend at the barrier
                f2 wl[5], wr[5], qL[5], qR[5];
#pragma unroll
                for (int f = 0; f < 5; f++) { wl[f] = wt[f * WTF + dl]; wr[f] = wt[f * WTF + dr]; }
#pragma unroll
                for (int f = 0; f < 5; f++) plm_m<MODE>(wl[f], W[f], wr[f], qL[f], qR[f]);
#pragma unroll
                for (int f = 0; f < 5; f++) {
                    if (cid == 1 && xact) sm.QLx[f][rp][0] = qL[f];   // column -1: left state of the tile's low x face
                    if (cid == 2 && xact) sm.QRxR[f][rp] = qR[f];     // column PTX: right state of the tile's high x face
                }
            }
            block_bar();
            // phase B: halo columns of plane k+1 (the flux through the tile's high x face is the producer warp's)
            if (k + 1 < kend) {
                mbar_wait_parity(&sm.full_halo[hs], hpar);
                const double* s = c0 + hs * CSLOT;
                float Wa[5], Wb[5];
                if (FBOX) {  // float boxes: [side][field][row][box column], 4 columns per box, 1280 bytes per side
                    const float* sf = reinterpret_cast<const float*>(&sm.hcol[0][0][0][0][0] + hs * CSLOT) +
                                      (cid >> 1) * (5 * PTY * 4) + (2 * rp) * 4 + bidx;
                    const float pref_f = (float)pref_d;
#pragma unroll
                    for (int f = 0; f < 5; f++) { Wa[f] = sf[f * PTY * 4]; Wb[f] = sf[f * PTY * 4 + 4]; }
                    if (SGL) {  // conserved fp32 state
                        float ca[5], cb[5];
#pragma unroll
                        for (int f = 0; f < 5; f++) { ca[f] = Wa[f]; cb[f] = Wb[f]; }
                        (void)recover(ca[0], ca[1], ca[2], ca[3], ca[4], (float)gm1, pref_f, rx, VN_KEEP, VN_KEEP, Wa);
                        (void)recover(cb[0], cb[1], cb[2], cb[3], cb[4], (float)gm1, pref_f, rx, VN_KEEP, VN_KEEP, Wb);
                    } else {    // float_t primitives of the van Leer predictor
                        Wa[1] = pdev(Wa[1], pref_f); Wb[1] = pdev(Wb[1], pref_f);
                        Wa[2] = apply_vn_rule(Wa[2], rx);  Wb[2] = apply_vn_rule(Wb[2], rx);
                    }
                } else {
                double ua[5], ub[5];
#pragma unroll
                for (int f = 0; f < 5; f++) { ua[f] = s[f * CF]; ub[f] = s[f * CF + 2]; }
                (void)recover(ua[0], ua[1], ua[2], ua[3], ua[4], (double)gm1, pref_d, rx, VN_KEEP, VN_KEEP, Wa);
                (void)recover(ub[0], ub[1], ub[2], ub[3], ub[4], (double)gm1, pref_d, rx, VN_KEEP, VN_KEEP, Wb);
                }
#pragma unroll
                for (int f = 0; f < 5; f++) {
                    W[f] = mk(Wa[f], Wb[f]);
                    if (xact) wt[f * WTF] = W[f];
                }
                if (++hs == NHALO) { hs = 0; hpar ^= 1u; }
            }
            block_bar();
        }
        block_bar();
    } else if (warp == WARP_PRODUCER) {
        // ================================ producer warp: all global traffic, by TMA =====================
        const HaloSide ylo = halo_side(j0 - 2, ny, g.bc[2], g.bc[3]);
        const HaloSide yhi = halo_side(j0 + PTY, ny, g.bc[2], g.bc[3]);
        constexpr int XW = FBOX ? 4 : 2;                               // halo column boxes: 2 doubles or 4 floats wide
        constexpr unsigned RAW_TX = FBOX ? OWN_BYTES / 2 : OWN_BYTES;  // float boxes are half the bytes
        constexpr unsigned HALO_TX = FBOX ? 4 * 1280 : 2 * ROW_BYTES + 2 * COL_BYTES;
        constexpr unsigned U0_TX = SGL ? OWN_BYTES / 2 : OWN_BYTES;
        const HaloSide xlo = halo_side(i0 - 2, nx, g.bc[0], g.bc[1], XW);
        const HaloSide xhi = halo_side(i0 + PTX, nx, g.bc[0], g.bc[1], XW);
        const int plast = kend + 2;  // planes up to kend+1 feed the z stencil; the main warps convert one plane further
                                     // (unconditionally: straight-line code), so that one is loaded too
        auto load_raw = [&](int p, int slot) {
            int rz;
            const int sk = bc_source(p, nz, g.bc[4], g.bc[5], rz);
            mbar_expect_tx(&sm.full_raw[slot], RAW_TX);
            // ghost planes of a communication boundary come from the array the neighbouring block has filled
            // (planes further out than two are loaded for the straight-line code only and never used)
            if (COMM && p < 0 && g.bc[4] == BC_COMM)
                tma_load4(&sm.raw[slot][0][0][0], &maps.in_glo, i0, j0, max(p + 2, 0), 0, &sm.full_raw[slot]);
            else if (COMM && p >= nz && g.bc[5] == BC_COMM)
                tma_load4(&sm.raw[slot][0][0][0], &maps.in_ghi, i0, j0, min(p - nz, 1), 0, &sm.full_raw[slot]);
            else
                tma_load4(&sm.raw[slot][0][0][0], &maps.in_own, i0, j0, sk, 0, &sm.full_raw[slot]);   // (slot stride follows the type)
        };
        // The updated plane p leaves by one TMA store; next to a communication boundary the same box is also stored into
        // the neighbouring block's ghost array over NVLink / peer memory: the halo exchange of Sec. 3.1.2 is part of the
        // stage kernel (no separate pack / send / unpack pass, no extra read of the state).
        auto store_plane = [&](int p, const void* src) {
            tma_store4(&maps.out_own, i0, j0, p, 0, src);
            if (COMM && g.bc[4] == BC_COMM && p < 2) tma_store4(&maps.out_plo, i0, j0, p, 0, src);
            if (COMM && g.bc[5] == BC_COMM && p >= nz - 2) tma_store4(&maps.out_phi, i0, j0, p - (nz - 2), 0, src);
            tma_commit();
        };
        auto load_halo = [&](int p, int slot) {  // p in [kbeg, kend): an interior plane
            unsigned long long* bar = &sm.full_halo[slot];
            mbar_expect_tx(bar, HALO_TX);
            // second side of each pair: right behind the first one (float boxes are 1280 bytes each)
            char* const r1 = FBOX ? reinterpret_cast<char*>(&sm.hrow[slot][0][0][0][0]) + 1280
                                         : reinterpret_cast<char*>(&sm.hrow[slot][1][0][0][0]);
            char* const c1 = FBOX ? reinterpret_cast<char*>(&sm.hcol[slot][0][0][0][0]) + 1280
                                         : reinterpret_cast<char*>(&sm.hcol[slot][1][0][0][0]);
            tma_load4(&sm.hrow[slot][0][0][0][0], &maps.in_rows, i0, ylo.start, p, 0, bar);
            tma_load4(r1, &maps.in_rows, i0, yhi.start, p, 0, bar);
            tma_load4(&sm.hcol[slot][0][0][0][0], &maps.in_cols, xlo.start, j0, p, 0, bar);
            tma_load4(c1, &maps.in_cols, xhi.start, j0, p, 0, bar);
        };
        if (lane == 0) {
            for (int q = 0; q < NSLOT; q++)
                if (pbase + q <= plast) load_raw(pbase + q, q);
            for (int m = 0; m < NHALO; m++)
                if (kbeg + m < kend) load_halo(kbeg + m, m);
        }
        int s_prev = 0;   // ring slot of plane k-1 (plane kbeg-2 at the first iteration)
        int hs = 0;       // halo slot of plane k (for k >= kbeg)
#pragma unroll 1
        for (int k = kfirst; k < kend; k++) {
            __syncwarp();
            block_bar();
            if (MODE == 2 && lane == 0) {
                // van Leer corrector: the primitive planes are only read, U^n is updated in place in the U0 ring
                const bool stored = k - 1 >= kbeg;
                if (k >= kbeg && k + NHALO < kend) load_halo(k + NHALO, hs);
                if (k - 1 + NSLOT <= plast) load_raw(k - 1 + NSLOT, s_prev);
                if (stored) store_plane(k - 1, &sm.u0[(k - 1 - kbeg) % NU0][0][0][0]);
                if (k + 1 < kend) {
                    const int m = (k + 1 - kbeg) % NU0;
                    // this slot held plane k-2, whose store was committed one group before the one just issued
                    if (stored) asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory");
                    mbar_expect_tx(&sm.full_u0[m], U0_TX);
                    tma_load4(&sm.u0[m][0][0][0], &maps.u0_own, i0, j0, k + 1, 0, &sm.full_u0[m]);
                }
            }
            if (MODE != 2 && lane == 0) {
                const bool stored = k - 1 >= kbeg;
                if (stored) store_plane(k - 1, &sm.raw[s_prev][0][0][0]);  // updated in place in phase C of the previous iteration
                if (k >= kbeg && k + NHALO < kend) load_halo(k + NHALO, hs);
                if (STAGE == 2 && k + 1 < kend) {
                    const int m = (k + 1 - kbeg) % NU0;
                    mbar_expect_tx(&sm.full_u0[m], U0_TX);
                    tma_load4(&sm.u0[m][0][0][0], &maps.u0_own, i0, j0, k + 1, 0, &sm.full_u0[m]);
                }
            }
            __syncwarp();
            if (MODE != 2 && lane == 0) {  // refill the slot the store is reading from
                const bool stored = k - 1 >= kbeg;
                const int p = k - 1 + NSLOT;
                if (p <= plast) {
                    if (stored) tma_wait_read0();  // the store has read the box: the slot may be refilled
                    load_raw(p, s_prev);
                }
            }
            if (++s_prev == NSLOT) s_prev = 0;
            if (k >= kbeg && ++hs == NHALO) hs = 0;
            __syncwarp();
            block_bar();
        }
        __syncwarp();
        block_bar();
        if (lane == 0) {  // the last plane of the slab
            if (MODE == 2) store_plane(kend - 1, &sm.u0[(kend - 1 - kbeg) % NU0][0][0][0]);
            else           store_plane(kend - 1, &sm.raw[s_prev][0][0][0]);
            tma_wait_all0();
        }
        __syncwarp();
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
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// cuTensorMapEncodeTiled through the runtime's driver entry point lookup (no link against libcuda)
inline EncodeTiledFn encode_tiled_fn()
{
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
    }
    return fn;
}

// Tensor map over one conserved state U[5][nz][ny][nx] (fp64, x fastest) with a box of bx x by x 1 x 5.
// nplanes: z extent of the array (the block's own, or 2 for the ghost arrays of a communication boundary).
inline bool make_map(CUtensorMap* m, const double* U, const Grid& g, int bx, int by, int nplanes = 0)
{
    EncodeTiledFn fn = encode_tiled_fn();
    if (!fn) return false;
    if (nplanes <= 0) nplanes = g.n[2];
    const cuuint64_t dims[4] = {(cuuint64_t)g.n[0], (cuuint64_t)g.n[1], (cuuint64_t)nplanes, 5};
    const cuuint64_t strides[3] = {(cuuint64_t)g.n[0] * 8, (cuuint64_t)g.n[0] * g.n[1] * 8,
                                   (cuuint64_t)g.n[0] * g.n[1] * nplanes * 8};
    const cuuint32_t box[4] = {(cuuint32_t)bx, (cuuint32_t)by, 1, 5};
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    return fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, (void*)U, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
              CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// Tensor map over a float_t primitive array W[5][nz][ny][nx] (van Leer predictor output), box bx x by x 1 x 5.
inline bool make_map_f32(CUtensorMap* m, const float* W, const Grid& g, int bx = PTX, int by = PTY)
{
    EncodeTiledFn fn = encode_tiled_fn();
    if (!fn) return false;
    const cuuint64_t dims[4] = {(cuuint64_t)g.n[0], (cuuint64_t)g.n[1], (cuuint64_t)g.n[2], 5};
    const cuuint64_t strides[3] = {(cuuint64_t)g.n[0] * 4, (cuuint64_t)g.n[0] * g.n[1] * 4, (cuuint64_t)g.N * 4};
    const cuuint32_t box[4] = {(cuuint32_t)bx, (cuuint32_t)by, 1, 5};
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    return fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, (void*)W, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
              CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

struct StageMaps;
inline void comm_defaults(StageMaps* sm);

// maps of both stages for the two state buffers of a handle: stage 1 reads A writes B, stage 2 reads B, averages with
// and writes A.
struct StageMaps {
    Maps s1, s2;
    bool ok;
};

// Without communication boundaries the four extra maps are never dereferenced; they alias the block's own arrays.
inline void comm_defaults(StageMaps* sm)
{
    sm->s1.in_glo = sm->s1.in_ghi = sm->s1.in_own; sm->s1.out_plo = sm->s1.out_phi = sm->s1.out_own;
    sm->s2.in_glo = sm->s2.in_ghi = sm->s2.in_own; sm->s2.out_plo = sm->s2.out_phi = sm->s2.out_own;
}

// Communication boundaries in z (Heun, fp64 state).  ghostA / ghostB [side]: this block's ghost arrays [5][2][ny][nx] of the
// state arrays A and B beyond its low (0) / high (1) z face; peerA / peerB [side]: the ghost arrays of the block beyond that
// face which hold THIS block's planes (its high-side ghosts for side 0, its low-side ghosts for side 1), addressable from
// this device (same process, or opened from a CUDA IPC handle).  NULL entries: that face is no communication boundary.
inline bool set_comm_maps(StageMaps* sm, const Grid& g, double* const ghostA[2], double* const ghostB[2],
                          double* const peerA[2], double* const peerB[2])
{
    CUtensorMap* in1[2] = {&sm->s1.in_glo, &sm->s1.in_ghi};
    CUtensorMap* in2[2] = {&sm->s2.in_glo, &sm->s2.in_ghi};
    CUtensorMap* out1[2] = {&sm->s1.out_plo, &sm->s1.out_phi};
    CUtensorMap* out2[2] = {&sm->s2.out_plo, &sm->s2.out_phi};
    for (int side = 0; side < 2; side++) {
        if (ghostA[side] && !make_map(in1[side], ghostA[side], g, PTX, PTY, 2)) return false;   // stage 1 reads A
        if (ghostB[side] && !make_map(in2[side], ghostB[side], g, PTX, PTY, 2)) return false;   // stage 2 reads B
        if (peerB[side] && !make_map(out1[side], peerB[side], g, PTX, PTY, 2)) return false;    // stage 1 writes B
        if (peerA[side] && !make_map(out2[side], peerA[side], g, PTX, PTY, 2)) return false;    // stage 2 writes A
    }
    return true;
}

inline bool supported(const Grid& g)
{
    return g.active[0] && g.active[1] && g.active[2] && g.n[0] % PTX == 0 && g.n[1] % PTY == 0 && g.n[2] >= 2 &&
           (g.N * 8) % 16 == 0 && (unsigned long long)g.N * 8 < (1ull << 40);
}

inline void build_maps(StageMaps* sm, const double* A, const double* B, const Grid& g)
{
    sm->ok = false;
    if (!supported(g)) return;
    CUtensorMap a_own, a_rows, a_cols, b_own, b_rows, b_cols;
    if (!make_map(&a_own, A, g, PTX, PTY) || !make_map(&a_rows, A, g, PTX, 2) || !make_map(&a_cols, A, g, 2, PTY) ||
        !make_map(&b_own, B, g, PTX, PTY) || !make_map(&b_rows, B, g, PTX, 2) || !make_map(&b_cols, B, g, 2, PTY))
        return;
    sm->s1.in_own = a_own; sm->s1.in_rows = a_rows; sm->s1.in_cols = a_cols; sm->s1.u0_own = a_own; sm->s1.out_own = b_own;
    sm->s2.in_own = b_own; sm->s2.in_rows = b_rows; sm->s2.in_cols = b_cols; sm->s2.u0_own = a_own; sm->s2.out_own = a_own;
    comm_defaults(sm);
    sm->ok = true;
}

// van Leer: the predictor reads the state A and writes the float_t primitives Wh (maps in sm->s1; s2 unused)
inline void build_maps_vl(StageMaps* sm, const double* A, const float* Wh, const Grid& g)
{
    sm->ok = false;
    if (!supported(g) || (g.N * 4) % 16 != 0) return;
    CUtensorMap a_own, a_rows, a_cols, w_own, w_rows, w_cols;
    if (!make_map(&a_own, A, g, PTX, PTY) || !make_map(&a_rows, A, g, PTX, 2) || !make_map(&a_cols, A, g, 2, PTY) ||
        !make_map_f32(&w_own, Wh, g) || !make_map_f32(&w_rows, Wh, g, PTX, 2) || !make_map_f32(&w_cols, Wh, g, 4, PTY))
        return;
    sm->s1.in_own = a_own; sm->s1.in_rows = a_rows; sm->s1.in_cols = a_cols; sm->s1.u0_own = a_own; sm->s1.out_own = w_own;
    // corrector: primitive planes and halo boxes from Wh (columns 4 floats = 16 bytes wide), U^n in and out through A
    sm->s2.in_own = w_own; sm->s2.in_rows = w_rows; sm->s2.in_cols = w_cols; sm->s2.u0_own = a_own; sm->s2.out_own = a_own;
    comm_defaults(sm);
    sm->ok = true;
}

// all-fp32 "Single" mode: both state arrays hold floats; stage 1 reads A writes B, stage 2 reads B, averages with and
// writes A.  Halo column boxes are 4 floats (16 bytes) wide.
inline void build_maps_single(StageMaps* sm, const float* A, const float* B, const Grid& g)
{
    sm->ok = false;
    if (!supported(g) || (g.N * 4) % 16 != 0) return;
    CUtensorMap a_own, a_rows, a_cols, b_own, b_rows, b_cols;
    if (!make_map_f32(&a_own, A, g) || !make_map_f32(&a_rows, A, g, PTX, 2) || !make_map_f32(&a_cols, A, g, 4, PTY) ||
        !make_map_f32(&b_own, B, g) || !make_map_f32(&b_rows, B, g, PTX, 2) || !make_map_f32(&b_cols, B, g, 4, PTY))
        return;
    sm->s1.in_own = a_own; sm->s1.in_rows = a_rows; sm->s1.in_cols = a_cols; sm->s1.u0_own = a_own; sm->s1.out_own = b_own;
    sm->s2.in_own = b_own; sm->s2.in_rows = b_rows; sm->s2.in_cols = b_cols; sm->s2.u0_own = a_own; sm->s2.out_own = a_own;
    comm_defaults(sm);
    sm->ok = true;
}

inline void launch_stage_single(int stage, const StageMaps& sm, const Grid& g, Ctrl* ctrl, int zchunk, cudaStream_t stream)
{
    dim3 grid(g.n[0] / PTX, g.n[1] / PTY, (g.n[2] + zchunk - 1) / zchunk);
    if (stage == 1) stage_tma<1, 0, float><<<grid, NTHREADS, sizeof(Smem<1, 0, float>) + 128, stream>>>(sm.s1, g, ctrl, zchunk);
    else            stage_tma<2, 0, float><<<grid, NTHREADS, sizeof(Smem<2, 0, float>) + 128, stream>>>(sm.s2, g, ctrl, zchunk);
}

inline void launch_vl_correct(const StageMaps& sm, const Grid& g, Ctrl* ctrl, int zchunk, cudaStream_t stream)
{
    dim3 grid(g.n[0] / PTX, g.n[1] / PTY, (g.n[2] + zchunk - 1) / zchunk);
    stage_tma<2, 2><<<grid, NTHREADS, sizeof(Smem<2, 2>) + 128, stream>>>(sm.s2, g, ctrl, zchunk);
}

inline void launch_vl_predict(const StageMaps& sm, const Grid& g, Ctrl* ctrl, int zchunk, cudaStream_t stream)
{
    dim3 grid(g.n[0] / PTX, g.n[1] / PTY, (g.n[2] + zchunk - 1) / zchunk);
    stage_tma<1, 1><<<grid, NTHREADS, sizeof(Smem<1>) + 128, stream>>>(sm.s1, g, ctrl, zchunk);
}

inline int auto_zchunk(const Grid& g)
{
    // >= ~6 waves of thread blocks over the SMs (148 on B200; the tail of the last wave costs ~1 %), slabs of >= 32 planes
    // (every slab converts two extra planes and primes its pipeline: ~3 planes of overhead)
    const long long tiles = (long long)(g.n[0] / PTX) * (g.n[1] / PTY);
    int chunk = g.n[2];
    while (chunk > 32 && tiles * ((g.n[2] + chunk - 1) / chunk) < (long long)sm_count() * BLOCKS_PER_SM * 6) chunk = (chunk + 1) / 2;
    return chunk;
}

inline void configure()
{
    constexpr size_t per_block = (228 * 1024) / BLOCKS_PER_SM - 1024;
    static_assert(sizeof(Smem<1>) + 128 <= per_block && sizeof(Smem<2>) + 128 <= per_block && sizeof(Smem<2, 2>) + 128 <= per_block,
                  "tile does not fit the shared memory of one SM");
    cudaFuncSetAttribute(stage_tma<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(Smem<1>) + 128);
    cudaFuncSetAttribute(stage_tma<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(Smem<2>) + 128);
    cudaFuncSetAttribute(stage_tma<2, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(Smem<2, 2>) + 128);
    cudaFuncSetAttribute(stage_tma<2, 2>, cudaFuncAttributePreferredSharedMemoryCarveout, (int)cudaSharedmemCarveoutMaxShared);
    cudaFuncSetAttribute(stage_tma<1, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(Smem<1>) + 128);
    cudaFuncSetAttribute(stage_tma<1, 1>, cudaFuncAttributePreferredSharedMemoryCarveout, (int)cudaSharedmemCarveoutMaxShared);
    cudaFuncSetAttribute(stage_tma<1>, cudaFuncAttributePreferredSharedMemoryCarveout, (int)cudaSharedmemCarveoutMaxShared);
    cudaFuncSetAttribute(stage_tma<2>, cudaFuncAttributePreferredSharedMemoryCarveout, (int)cudaSharedmemCarveoutMaxShared);
    cudaFuncSetAttribute(stage_tma<1, 0, double, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(Smem<1>) + 128);
    cudaFuncSetAttribute(stage_tma<2, 0, double, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(Smem<2>) + 128);
    cudaFuncSetAttribute(stage_tma<1, 0, double, true>, cudaFuncAttributePreferredSharedMemoryCarveout, (int)cudaSharedmemCarveoutMaxShared);
    cudaFuncSetAttribute(stage_tma<2, 0, double, true>, cudaFuncAttributePreferredSharedMemoryCarveout, (int)cudaSharedmemCarveoutMaxShared);
    cudaFuncSetAttribute(stage_tma<1, 0, float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(Smem<1, 0, float>) + 128);
    cudaFuncSetAttribute(stage_tma<2, 0, float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(Smem<2, 0, float>) + 128);
    cudaFuncSetAttribute(stage_tma<1, 0, float>, cudaFuncAttributePreferredSharedMemoryCarveout, (int)cudaSharedmemCarveoutMaxShared);
    cudaFuncSetAttribute(stage_tma<2, 0, float>, cudaFuncAttributePreferredSharedMemoryCarveout, (int)cudaSharedmemCarveoutMaxShared);
}

inline void launch_stage(int stage, const StageMaps& sm, const Grid& g, Ctrl* ctrl, int zchunk, cudaStream_t stream)
{
    dim3 grid(g.n[0] / PTX, g.n[1] / PTY, (g.n[2] + zchunk - 1) / zchunk);
    const bool comm = g.bc[4] == BC_COMM || g.bc[5] == BC_COMM;
    if (comm && stage == 1) stage_tma<1, 0, double, true><<<grid, NTHREADS, sizeof(Smem<1>) + 128, stream>>>(sm.s1, g, ctrl, zchunk);
    else if (comm)          stage_tma<2, 0, double, true><<<grid, NTHREADS, sizeof(Smem<2>) + 128, stream>>>(sm.s2, g, ctrl, zchunk);
    else if (stage == 1)    stage_tma<1><<<grid, NTHREADS, sizeof(Smem<1>) + 128, stream>>>(sm.s1, g, ctrl, zchunk);
    else                    stage_tma<2><<<grid, NTHREADS, sizeof(Smem<2>) + 128, stream>>>(sm.s2, g, ctrl, zchunk);
}

}  // namespace tma
}  // namespace kh
