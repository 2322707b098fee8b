// kh_strip.cuh -- KRATOS_KERNEL_STRIP: the fused stage kernel of 2D blocks (x and y active, nz == 1) in mixed
// precision (float_t = fp32, float2_t = fp64) and in the all-fp32 "Single" mode (float2_t = fp32,
// PAPER.md:240; the mode of the paper's 2D performance table): one warp = one independent pipeline.
//
// A warp owns a strip of SW = 28 columns and marches along y through a slab of rows, two rows per trip:
//   * lane l holds column x0 - 2 + l of the strip's 32-column window; the two outer lanes on either side are the
//     2-cell halo of the PLM stencil and are recomputed by the neighbouring strip (28 of 32 lanes produce output),
//     so every x neighbour of a cell lives in the neighbouring LANE: slopes, left states and fluxes cross the strip
//     by warp shuffles, and a warp never waits for another warp -- no block barrier anywhere in the kernel;
//   * a thread holds the row pair (2p, 2p+1) packed as f32x2, like the 3D kernels hold (2w, 2w+1): the slopes of
//     Eq. 3 and the HLLC solver of Eq. 4-5 run on packed FADD2 / FMUL2 / FFMA2, the x faces and the y faces of the pair
//     in lock step (tma::hllc2n<2>).  The y face between the two rows is internal to the thread; the face below the
//     pair was solved one trip earlier and the one above it is solved one trip later, so the march carries the
//     limited state of the last row and the fp64 flux sum of the pair, and the pair is updated one trip after it was
//     solved: the y direction lives in registers, as z does in the 3D kernels;
//   * global -> shared traffic is one TMA box (32 x 2 x 5 doubles) per row pair and warp, prefetched three pairs ahead
//     into a ring of NRING slots, completing on the warp's own mbarriers; at the domain edge two extra 2-column boxes
//     bring the ghost columns from where the boundary rule of Sec. 3.1.1 takes them (periodic wrap,
//     clamp, mirror), and ghost rows are a choice of box coordinates, exactly as in kh_tma.cuh;
//   * the update is fp64: raw state from the ring + flux sums, Heun average with U0 (cp.async
//     copies of the lane's own column, issued one trip ahead), coalesced 8-byte stores; stage 2 reduces the CFL rate of the new state
//     (PAPER.md:173).
// Warps are independent, so their load, convert, solve and update phases interleave on the SM by themselves; 12 warps
// per SM (three blocks of four warps).
//
// Bit-identical fluxes across strip and slab seams: both copies of a shared face run the same explicitly rounded
// operations (kh_pair.cuh) on the same inputs, so the fp64 contributions cancel exactly.
#pragma once
#include "kh_tma.cuh"

namespace kh {
namespace strip {

using pr::f2;
using pr::mk;
using pr::plm;
using pr::recover;
using pr::Gas;
using tma::HaloSide;
using tma::halo_side;

constexpr int SW = 28;        // columns of output per warp (lanes 2..29 of the 32-lane window)
constexpr int NRING = 5;      // row pairs in flight per warp: p-1 (update), p, p+1 (converted ahead), p+2, p+3 (arriving)
#ifndef KH_STRIP_WARPS
#define KH_STRIP_WARPS 4
#endif
#ifndef KH_STRIP_BLOCKS
#define KH_STRIP_BLOCKS 3
#endif
constexpr int WARPS = KH_STRIP_WARPS;           // warps per block (independent of each other)
constexpr int BLOCKS_PER_SM = KH_STRIP_BLOCKS;  // 12 warps per SM at <= 168 registers
constexpr unsigned HBOX_BYTES = 160;   // a ghost-column box: 5 fields x 2 rows x 16 bytes (2 doubles or 4 floats)

// ST = float2_t, the type the conserved state is stored in: double, or float in the all-fp32 "Single" mode.
// The box of a row pair starts on a 16-byte boundary of global memory (a box of floats starting 8 bytes off one raised
// "illegal instruction" on sm_100a): doubles x0 - 2, 32 wide; floats x0 - 4, 36 wide, the lane's column two elements in.
template <typename ST> struct Box { static constexpr int W = 32, OFF = 0; };
template <> struct Box<float> { static constexpr int W = 36, OFF = 2; };

template <typename ST>
struct WarpSmem {
    struct alignas(128) Slot { ST v[5][2][Box<ST>::W]; };
    Slot raw[NRING];                             // TMA box of a row pair: [field][row][column]
    alignas(128) unsigned char hx[NRING][2][256];  // ghost-column boxes [side]: [5 fields][2 rows][16 bytes], padded to 256 B
    alignas(16) ST u0[5][2][32];                 // stage 2: U0 of the two rows the NEXT trip updates; every lane copies and reads
                                                 // its own column only (cp.async), so the slot needs no second buffer
    unsigned long long full[NRING];
};

struct Maps {
    CUtensorMap in_own, in_cols;   // stage input: 32 x 2 x 5 box, 2 x 2 x 5 box
};

__device__ __forceinline__ void tma_load3(void* dst, const CUtensorMap* map, int c0, int c1, int c2, unsigned long long* bar)
{
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::
            "r"(tma::smem_u32(dst)), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(tma::smem_u32(bar))
        : "memory");
}

__device__ __forceinline__ f2 shfl_up2(f2 v)
{
    return mk(__shfl_up_sync(0xffffffffu, v.x, 1), __shfl_up_sync(0xffffffffu, v.y, 1));
}
__device__ __forceinline__ f2 shfl_down2(f2 v)
{
    return mk(__shfl_down_sync(0xffffffffu, v.x, 1), __shfl_down_sync(0xffffffffu, v.y, 1));
}

// One Heun stage of a 2D block.  STAGE 1: Uout = Uin + dt L(Uin).  STAGE 2: Uout = 1/2 U0 + 1/2 (Uin +
// dt L(Uin)) (Uout aliases U0) and the CFL rate maximum of Uout.
// rows_per_slab is even; a warp handles strip (id % nstrips), slab (id / nstrips).
template <int STAGE, typename ST = double>
__global__ void __launch_bounds__(WARPS * 32, BLOCKS_PER_SM)
stage_strip(const __grid_constant__ Maps maps, const ST* U0, ST* Uout, Grid g, Ctrl* ctrl, int rows_per_slab,
            int nstrips, int nwork)
{
    constexpr bool SGL = sizeof(ST) == 4;          // all-fp32 state: float boxes, fp32 recovery and update, no reference pressure
    constexpr int XW = SGL ? 4 : 2;                // columns of a ghost-column box (16 bytes)
    constexpr int BW = Box<ST>::W;                 // columns of the row-pair box
    constexpr int SLOT = sizeof(typename WarpSmem<ST>::Slot) / sizeof(ST);   // element stride of the ring
    constexpr unsigned BOX_BYTES = 5 * 2 * BW * sizeof(ST);
    using ST2 = typename std::conditional<SGL, float2, double2>::type;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    WarpSmem<ST>& sm = reinterpret_cast<WarpSmem<ST>*>(smem_raw)[warp];

    const double dt = ctrl->dt;
    if (!(dt > 0.0)) return;  // a step clipped to zero length (run_until past t_end) does nothing
    const int work = blockIdx.x * WARPS + warp;
    if (work >= nwork) return;   // (whole warps: no block-wide synchronisation exists in this kernel)
    const double pref_d = SGL ? 0.0 : ctrl->p_ref;
    const int nx = g.n[0], ny = g.n[1];
    const long long N = g.N;
    const int s = work % nstrips, slab = work / nstrips;
    const int x0 = s * SW;                         // first output column
    const int c = x0 - 2 + lane;                   // this lane's column
    const int npair = ny / 2;
    const int pbeg = slab * (rows_per_slab / 2);
    const int pend = min(pbeg + rows_per_slab / 2, npair);   // pairs [pbeg, pend)
    const ST gm1 = ST(g.gamma - 1.0);
    const ST pref_s = ST(pref_d);
    Gas gas;
    gas.gamma = (float)g.gamma;
    gas.g1 = (float)((g.gamma + 1.0) / (2.0 * g.gamma));
    gas.igm1 = (float)(1.0 / (g.gamma - 1.0));
    gas.pref = (float)pref_d;

    // ---- where this lane's column comes from (Sec. 3.1.1 in x) ----
    // interior column: the strip's own box.  Ghost column (c in {-2,-1} or {nx, nx+1}): one of the two ghost boxes.
    const HaloSide xlo = halo_side(-2, nx, g.bc[0], g.bc[1], XW);
    const HaloSide xhi = halo_side(nx, nx, g.bc[0], g.bc[1], XW);
    const bool ghost_lo = c < 0, ghost_hi = c >= nx && c < nx + 2;
    const bool need_lo = x0 - 2 < 0, need_hi = x0 - 2 + 32 > nx;      // warp-uniform: this strip touches a domain edge
    const int rx = ghost_lo ? xlo.rule : (ghost_hi ? xhi.rule : VN_KEEP);
    const int hx_idx = ghost_lo ? ((c == -2) ? xlo.idx0 : xlo.idx1) : ((c == nx) ? xhi.idx0 : xhi.idx1);
    const bool owner = lane >= 2 && lane < 2 + SW && c < nx;          // this lane's cells are written by this warp
    // element offsets of this lane inside a ring slot: own box [field][row][32], ghost box [side][field][row][2]
    const ST* const own_base = &sm.raw[0].v[0][0][lane + Box<ST>::OFF];
    const ST* const hx_base = reinterpret_cast<const ST*>(&sm.hx[0][ghost_hi ? 1 : 0][0]) + hx_idx;
    const bool from_ghost_box = ghost_lo || ghost_hi;

    if (lane == 0) {
        for (int q = 0; q < NRING; q++) mbar_init(&sm.full[q], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncwarp();

    // pair q (rows 2q, 2q+1; q in [-1, npair]) -> the box rows that hold it (Sec. 3.1.1 in y).  Interior pairs are
    // their own source; the two ghost pairs of the block take theirs from where the boundary rule says.
    const HaloSide ylo = halo_side(-2, ny, g.bc[2], g.bc[3]);
    const HaloSide yhi = halo_side(ny, ny, g.bc[2], g.bc[3]);
    const unsigned tx_bytes = BOX_BYTES + (need_lo ? HBOX_BYTES : 0u) + (need_hi ? HBOX_BYTES : 0u);
    auto issue = [&](int q, int slot) {   // lane 0
        const int row = (q < 0) ? ylo.start : ((q >= npair) ? yhi.start : 2 * q);
        unsigned long long* bar = &sm.full[slot];
        tma::mbar_expect_tx(bar, tx_bytes);
        tma_load3(&sm.raw[slot].v[0][0][0], &maps.in_own, x0 - 2 - Box<ST>::OFF, row, 0, bar);
        if (need_lo) tma_load3(&sm.hx[slot][0][0], &maps.in_cols, xlo.start, row, 0, bar);
        if (need_hi) tma_load3(&sm.hx[slot][1][0], &maps.in_cols, xhi.start, row, 0, bar);
    };
    // Each slot's mbarrier flips once per use: bit `slot` of phase_bits is the parity to wait for next.
    unsigned phase_bits = 0u;
    int hits = 0;
    auto convert = [&](int q, int slot, f2 (&W)[5], bool count) {
        int i0 = 0, i1 = 1, ry = VN_KEEP;
        if (q < 0) { i0 = ylo.idx0; i1 = ylo.idx1; ry = ylo.rule; }
        else if (q >= npair) { i0 = yhi.idx0; i1 = yhi.idx1; ry = yhi.rule; }
        tma::mbar_wait_parity(&sm.full[slot], (phase_bits >> slot) & 1u);
        phase_bits ^= 1u << slot;
        ST ua[5], ub[5];
        if (from_ghost_box) {
            const ST* b = hx_base + slot * (2 * 256 / (int)sizeof(ST));
#pragma unroll
            for (int f = 0; f < 5; f++) { ua[f] = b[f * 2 * XW + i0 * XW]; ub[f] = b[f * 2 * XW + i1 * XW]; }
        } else {
            const ST* b = own_base + slot * SLOT;
#pragma unroll
            for (int f = 0; f < 5; f++) { ua[f] = b[f * 2 * BW + i0 * BW]; ub[f] = b[f * 2 * BW + i1 * BW]; }
        }
        float Wa[5], Wb[5];
        const int ha = recover(ua[0], ua[1], ua[2], ua[3], ua[4], gm1, pref_s, rx, ry, VN_KEEP, Wa);
        const int hb = recover(ub[0], ub[1], ub[2], ub[3], ub[4], gm1, pref_s, rx, ry, VN_KEEP, Wb);
        if (count && owner) hits += ha + hb;
#pragma unroll
        for (int f = 0; f < 5; f++) W[f] = mk(Wa[f], Wb[f]);
    };

    // ---- prologue: pairs pbeg-1 .. pbeg+2 in flight (slots 0..3), W(pbeg-1) and W(pbeg) converted ----
    if (lane == 0)
        for (int q = pbeg - 1; q <= min(pbeg + 2, pend); q++) issue(q, q - (pbeg - 1));
    f2 WA[5], WB[5];              // W(p) and W(p+1), swapping roles from trip to trip
    float Wmy[5];                 // upper row of pair p-1
    float QLc[5];                 // left state of the y face below row 2p (limited state of row 2p-1 at its upper face)
    ST pend_y[5];                 // flux sum of row 2p-1, lacking the face above it (which trip p solves)
    {
        f2 Wm[5];
        convert(pbeg - 1, 0, Wm, false);
        convert(pbeg, 1, WA, true);
#pragma unroll
        for (int f = 0; f < 5; f++) {
            f2 qL, qR;
            plm(mk(Wm[f].x, Wm[f].x), Wm[f], mk(Wm[f].y, WA[f].x), qL, qR);   // row 2pbeg-1 from rows 2pbeg-2, 2pbeg-1, 2pbeg
            QLc[f] = qL.y;
            Wmy[f] = Wm[f].y;
            pend_y[f] = ST(0);
        }
    }
    const ST dtdx = ST(dt * g.inv_dx[0]), dtdy = ST(dt * g.inv_dx[1]);
    const CflConst<float> cc(g);
    f2 rate = mk(0.0f, 0.0f);
    const long long col_off = (long long)(owner ? c : 0);
    // ring slots of the pairs p-1 (row 2p-1 updated), p+1 (converted) and p+3 (issued) at trip p; pair p sits in s_upd + 1
    int s_upd = 0, s_conv = 2, s_issue = 4;
    // U0 of rows 2p-1 and 2p (the rows trip p updates), fetched one trip ahead: 8-byte cp.async copies of the lane's own
    // column into its own entries of sm.u0, a whole trip of latency hidden (the plain loads of the first version, issued and
    // consumed in the same trip, cost stage 2 two stalled cycles per issued one: round-2 capture r2a, profiles/history.md: long_sb)
    auto fetch_u0 = [&](int p) {
        if (STAGE != 2) return;
        const bool a = (p > pbeg) && owner, b = (p < pend) && owner;
        const long long cell = (long long)(2 * p - 1) * nx + col_off;
        ST* d = &sm.u0[0][0][lane];
#pragma unroll
        for (int f = 0; f < 5; f++) {
            if (a) __pipeline_memcpy_async(d + f * 64, U0 + f * N + cell, sizeof(ST));
            if (b) __pipeline_memcpy_async(d + f * 64 + 32, U0 + f * N + cell + nx, sizeof(ST));
        }
        __pipeline_commit();
    };
    fetch_u0(pbeg);

    // Trip p solves the faces of pair p; that completes row 2p-1 (the face above it was missing) and row 2p, which are
    // updated and stored; row 2p+1 waits for the next trip.  The first trip of a slab stores row 2p only, the last one
    // (p == pend) row 2p-1 only.  W0 = W(p) on entry, Wp receives W(p+1).
    auto trip = [&](int p, f2 (&W0)[5], f2 (&Wp)[5]) {
        if (lane == 0 && p + 3 <= pend) issue(p + 3, s_issue);    // into the slot pair p-2 left in trip p-1
        const bool upd_a = (p > pbeg) && owner, upd_b = (p < pend) && owner;   // rows 2p-1, 2p
        const long long cell_a = (long long)(2 * p - 1) * nx + col_off;        // row 2p-1; row 2p is + nx
        if (p + 1 <= pend) convert(p + 1, s_conv, Wp, p + 1 < pend);
        // ---- slopes (Eq. 3) and the two face pairs of pair p ----
        f2 L[2][5], R[2][5], Fn[2][5];
        {
            f2 qLx[5], qRx[5], qLy[5], qRy[5];
#pragma unroll
            for (int f = 0; f < 5; f++) {
                const f2 xm = shfl_up2(W0[f]), xp = shfl_down2(W0[f]);
                plm(xm, W0[f], xp, qLx[f], qRx[f]);
                pr::plm_along_pair(Wmy[f], W0[f], Wp[f].x, qLy[f], qRy[f]);
                Wmy[f] = W0[f].y;
            }
            f2 t[5];
#pragma unroll
            for (int f = 0; f < 5; f++) t[f] = shfl_up2(qLx[f]);           // left state of the face at c - 1/2
            tma::to_normal<0>(t, L[0]);
            tma::to_normal<0>(qRx, R[0]);
#pragma unroll
            for (int f = 0; f < 5; f++) { t[f] = mk(QLc[f], qLy[f].x); QLc[f] = qLy[f].y; }   // faces 2p-1/2, 2p+1/2
            tma::to_normal<1>(t, L[1]);
            tma::to_normal<1>(qRy, R[1]);
        }
        tma::hllc2n<2>(L, R, gas, Fn);
        // U0 of the two rows for the Heun average (fetched during the previous trip); the next trip's fetch follows at once
        ST2 v0[5];
        if (STAGE == 2) {
            __pipeline_wait_prior(0);
            const ST* d = &sm.u0[0][0][lane];
#pragma unroll
            for (int f = 0; f < 5; f++) { v0[f].x = d[f * 64]; v0[f].y = d[f * 64 + 32]; }   // (rows not updated: stale, unused)
            if (p + 1 <= pend) fetch_u0(p + 1);
        }
        ST ua[5], ub[5];   // new state of rows 2p-1, 2p
        {
            f2 Fx[5], Fy[5];
            tma::from_normal<0>(Fn[0], Fx);
            tma::from_normal<1>(Fn[1], Fy);
            const ST* ba = own_base + s_upd * SLOT + BW;                                       // row 2p-1 in the ring
            const ST* bb = own_base + ((s_upd + 1 == NRING) ? 0 : s_upd + 1) * SLOT;   // row 2p
#pragma unroll
            for (int f = 0; f < 5; f++) {
                const f2 fxh = shfl_down2(Fx[f]);                          // flux through the face at c + 1/2
                const ST flo = (ST)Fy[f].x, fin = (ST)Fy[f].y;
                // fp64 update.  Row 2p-1: its sum so far and the face above it (2p-1/2).
                // Row 2p: x faces, y faces 2p-1/2 (+) and 2p+1/2 (-).  Row 2p+1 so far: x faces, y face 2p+1/2 (+).
                ST xa = add_(ba[f * 2 * BW], fma_(-dtdy, flo, pend_y[f]));
                ST xb = add_(bb[f * 2 * BW], fma_(dtdy, sub_(flo, fin), mul_(dtdx, sub_((ST)Fx[f].x, (ST)fxh.x))));
                pend_y[f] = fma_(dtdy, fin, mul_(dtdx, sub_((ST)Fx[f].y, (ST)fxh.y)));
                if (STAGE == 2) {
                    xa = fma_(ST(0.5), v0[f].x, mul_(ST(0.5), xa));
                    xb = fma_(ST(0.5), v0[f].y, mul_(ST(0.5), xb));
                }
                ua[f] = xa;
                ub[f] = xb;
                if (upd_a) Uout[f * N + cell_a] = xa;
                if (upd_b) Uout[f * N + cell_a + nx] = xb;
            }
        }
        {
            if (STAGE == 2) {   // CFL rate of the new state (readings S1/S7), both rows at once
                using namespace pr;
                const float rfl = (float)KH_RHO_FLOOR, pfl = (float)KH_P_FLOOR;
                f2 r = mk((float)ua[0], (float)ub[0]);
                r = mk(r.x < rfl ? rfl : r.x, r.y < rfl ? rfl : r.y);  // comparisons, not fmax: a NaN must survive
                const f2 ir = rcp2(r);
                const f2 vx = mul2(mk((float)ua[1], (float)ub[1]), ir);
                const f2 vy = mul2(mk((float)ua[2], (float)ub[2]), ir);
                const f2 vz = mul2(mk((float)ua[3], (float)ub[3]), ir);
                const f2 v2 = fma2(vz, vz, fma2(vy, vy, mul2(vx, vx)));
                f2 pp = mul2(bc(cc.gm1), fma2(mul2(bc(-0.5f), r), v2, mk((float)ua[4], (float)ub[4])));
                pp = mk(pp.x < pfl ? pfl : pp.x, pp.y < pfl ? pfl : pp.y);
                const f2 gp = mul2(bc(cc.gamma), pp);
                const f2 cs = mul2(gp, rsqrt2(mul2(gp, r)));
                f2 rt = mul2(add2(mk(fabsf(vx.x), fabsf(vx.y)), cs), bc(cc.idx));
                rt = fma2(add2(mk(fabsf(vy.x), fabsf(vy.y)), cs), bc(cc.idy), rt);
                if (!(rt.x == rt.x)) rt.x = __int_as_float(0x7f800000);
                if (!(rt.y == rt.y)) rt.y = __int_as_float(0x7f800000);
                rate = mk(upd_a ? fmaxf(rate.x, rt.x) : rate.x, upd_b ? fmaxf(rate.y, rt.y) : rate.y);
            }
        }
        __syncwarp();   // every lane has read pair p-1 from the ring before lane 0 refills that slot in the next trip
        if (++s_upd == NRING) s_upd = 0;
        if (++s_conv == NRING) s_conv = 0;
        if (++s_issue == NRING) s_issue = 0;
    };
#pragma unroll 1
    for (int p = pbeg; p <= pend; p += 2) {   // two trips per turn: the two register sets swap roles instead of being copied
        trip(p, WA, WB);
        if (p + 1 <= pend) trip(p + 1, WB, WA);
    }

    if (hits) atomicAdd(&ctrl->floor_hits, (unsigned long long)hits);
    if (STAGE == 2) {
        float r = fmaxf(rate.x, rate.y);
        for (int o = 16; o > 0; o >>= 1) r = fmaxf(r, __shfl_xor_sync(0xffffffffu, r, o));
        if (lane == 0 && r > 0.0f) atomicMax(&ctrl->rate_bits, (unsigned long long)__double_as_longlong((double)r));
    }
}

// ---------------------------------------------------------------------------------------
// host side
inline bool supported(const Grid& g)
{
    return g.active[0] && g.active[1] && !g.active[2] && g.n[0] % 2 == 0 && g.n[1] % 2 == 0 && g.n[0] >= 4 && g.n[1] >= 4;
}

// all-fp32 "Single" mode: float boxes need 16-byte row strides
inline bool supported_single(const Grid& g) { return supported(g) && g.n[0] % 4 == 0; }

// Tensor map over the 2D state U[5][ny][nx] (x fastest; doubles or floats) with a box of bx x 2 x 5.
template <typename ST>
inline bool make_map(CUtensorMap* m, const ST* U, const Grid& g, int bx)
{
    tma::EncodeTiledFn fn = tma::encode_tiled_fn();
    if (!fn) return false;
    const cuuint64_t dims[3] = {(cuuint64_t)g.n[0], (cuuint64_t)g.n[1], 5};
    const cuuint64_t strides[2] = {(cuuint64_t)g.n[0] * sizeof(ST), (cuuint64_t)g.N * sizeof(ST)};
    const cuuint32_t box[3] = {(cuuint32_t)bx, 2, 5};
    const cuuint32_t estr[3] = {1, 1, 1};
    return fn(m, sizeof(ST) == 4 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, (void*)U, dims, strides, box,
              estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

struct StageMaps {
    Maps s1, s2;   // stage 1 reads A, stage 2 reads B
    bool ok;
};

// ghost-column boxes are 16 bytes wide: 2 doubles or 4 floats
template <typename ST>
inline void build_maps(StageMaps* sm, const ST* A, const ST* B, const Grid& g)
{
    sm->ok = false;
    if (sizeof(ST) == 4 ? !supported_single(g) : !supported(g)) return;
    const int xw = 16 / (int)sizeof(ST);
    if (!make_map(&sm->s1.in_own, A, g, Box<ST>::W) || !make_map(&sm->s1.in_cols, A, g, xw) ||
        !make_map(&sm->s2.in_own, B, g, Box<ST>::W) || !make_map(&sm->s2.in_cols, B, g, xw))
        return;
    sm->ok = true;
}

inline int auto_rows(const Grid& g)
{
    // One wave of equal work items: every SM holds BLOCKS_PER_SM x WARPS warps, each marching through one slab from
    // the start of the kernel to its end, so that the prologue of a slab (two extra row pairs converted, the first box
    // awaited) is paid once per warp.  Slabs shorter than 16 rows are not worth their prologue: small blocks then
    // simply leave SMs idle (they are launch-bound anyway).
    const long long nstrips = (g.n[0] + SW - 1) / SW;
    const long long slots = (long long)sm_count() * WARPS * BLOCKS_PER_SM;
    long long nslabs = slots / nstrips;
    if (nslabs < 1) nslabs = 1;
    int rows = (int)((g.n[1] + nslabs - 1) / nslabs);
    rows = (rows + 1) & ~1;
    if (rows < 16) rows = 16;
    return rows < g.n[1] ? rows : g.n[1];
}

template <typename ST>
inline void configure_for()
{
    cudaFuncSetAttribute(stage_strip<1, ST>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(WARPS * sizeof(WarpSmem<ST>)));
    cudaFuncSetAttribute(stage_strip<2, ST>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(WARPS * sizeof(WarpSmem<ST>)));
    cudaFuncSetAttribute(stage_strip<1, ST>, cudaFuncAttributePreferredSharedMemoryCarveout, (int)cudaSharedmemCarveoutMaxShared);
    cudaFuncSetAttribute(stage_strip<2, ST>, cudaFuncAttributePreferredSharedMemoryCarveout, (int)cudaSharedmemCarveoutMaxShared);
}
inline void configure()
{
    configure_for<double>();
    configure_for<float>();
}

template <typename ST>
inline void launch_stage(int stage, const StageMaps& sm, const ST* U0, ST* Uout, const Grid& g, Ctrl* ctrl, int rows,
                         cudaStream_t stream)
{
    rows = (rows + 1) & ~1;
    const int nstrips = (g.n[0] + SW - 1) / SW;
    const int nslabs = (g.n[1] + rows - 1) / rows;
    const int nwork = nstrips * nslabs;
    const unsigned blocks = (unsigned)((nwork + WARPS - 1) / WARPS);
    const size_t smem = WARPS * sizeof(WarpSmem<ST>);
    if (stage == 1) stage_strip<1, ST><<<blocks, WARPS * 32, smem, stream>>>(sm.s1, U0, Uout, g, ctrl, rows, nstrips, nwork);
    else            stage_strip<2, ST><<<blocks, WARPS * 32, smem, stream>>>(sm.s2, U0, Uout, g, ctrl, rows, nstrips, nwork);
}

}  // namespace strip
}  // namespace kh
