/*
 * kratos_oracle.c -- ORACLE.  TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * A plain, slow, all-fp64 CPU restatement of the hydrodynamic hot path of
 *   L. Wang, "The Kratos Framework for Heterogeneous Astrophysical Simulations:
 *   Fundamental Infrastructures and Hydrodynamics" (arXiv 2501.02317),
 * written from the text of the paper only.  Citations are
 * "PAPER.md:<line>" plus the section / equation.  Readings of points on which the
 * paper is silent (S1..S11) are the ones listed in DESIGN.md section 3.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may load this file.  It shares no code with the CUDA path (no common header,
 * helper or constant) and the CUDA path never calls it.
 *
 * Layout: conserved state U = (rho, m_x, m_y, m_z, eps), struct-of-arrays
 * [5][nz][ny][nx], x fastest, interior cells only.  An axis is "active" when its
 * extent is > 1; inactive axes carry no ghosts and no flux.
 *
 * Pinned by tests/test_oracle_pins.py (exact Riemann solution, advected density wave
 * with the paper's N^-2 order, exact conservation, uniform-state fixed point,
 * stationary/moving contact, consistency, axis interchange / mirror, monotonicity,
 * independent brute force).  Parity UNPINNED for: Kratos' own (unpublished) choice of
 * CFL formula (S1), of the p* estimate entering Eq. 5 (S3), of floors (S6) and of the
 * van Leer integrator's sub-steps (S15, orc_step_vl) -- no output of the real code exists
 * to compare against.
 *
 * No blocking, fusion or reordering beyond what the paper's algorithm states; the
 * only concession to speed is "#pragma omp parallel for" on outermost loops, which
 * does not change any arithmetic.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>

#define NGH 2 /* PLM is 2nd order => 2 ghost layers (Sec. 3.1) */

#define ORC_RHO_FLOOR 1e-30 /* reading S6 */
#define ORC_P_FLOOR 1e-30   /* reading S6 */

/* boundary codes, in the order of the paper's list */
enum { BC_PERIODIC = 0, BC_FREE = 1, BC_OUTFLOW = 2, BC_REFLECT = 3 };

/* primitive slots: the paper's set (rho, p, v) */
enum { IR = 0, IP = 1, IVX = 2, IVY = 3, IVZ = 4 };

/* ------------------------------------------------------------------------- */
/* Eq. 3: minmod.  The printed cases omit ab = 0; reading S2: 0. */
double orc_minmod(double a, double b)
{
    if (a * b > 0.0) {
        if (fabs(a) < fabs(b)) return a;
        return b;
    }
    return 0.0;
}

/* ------------------------------------------------------------------------- */
/* Sec. 3.1: conservative -> primitive, with eps = eps_g + rho v^2/2
 * and the ideal-gas closure p = (gamma-1) eps_g.  Floors act on the
 * primitives only (S6); *hits counts activations.  Returns nothing; W = (rho,p,vx,vy,vz). */
void orc_cons_to_prim(const double U[5], double gamma, double W[5], long long *hits)
{
    double rho = U[0];
    if (rho < ORC_RHO_FLOOR) { rho = ORC_RHO_FLOOR; if (hits) (*hits)++; }
    double vx = U[1] / rho, vy = U[2] / rho, vz = U[3] / rho;
    double ekin = 0.5 * (U[1] * U[1] + U[2] * U[2] + U[3] * U[3]) / rho;
    double p = (gamma - 1.0) * (U[4] - ekin);
    if (p < ORC_P_FLOOR) { p = ORC_P_FLOOR; if (hits) (*hits)++; }
    W[IR] = rho; W[IP] = p; W[IVX] = vx; W[IVY] = vy; W[IVZ] = vz;
}

/* ------------------------------------------------------------------------- */
/* Sec. 3.2.2: HLLC flux across a face whose normal is the local
 * "x".  WL, WR = (rho, p, u, v, w) with u normal and v, w tangential.
 * F = (mass, normal momentum, tangential momentum 1, tangential momentum 2, energy).
 *   Eq. 5: Delta s_L = -c_L q_L, Delta s_R = +c_R q_R,
 *          q_K = sqrt(1 + (gamma+1)/(2 gamma) (max(p_star/p_K, 1) - 1));
 *   p_star: reading S3 (acoustic / primitive-variable estimate, floored at 0);
 *   Eq. 4: contact speed s_star written with Delta s_K;
 *   star states / flux selection: reading S4 (standard HLLC assembly). */
void orc_hllc(const double WL[5], const double WR[5], double gamma, double F[5])
{
    const double rL = WL[0], pL = WL[1], uL = WL[2], vL = WL[3], wL = WL[4];
    const double rR = WR[0], pR = WR[1], uR = WR[2], vR = WR[3], wR = WR[4];

    const double cL = sqrt(gamma * pL / rL);
    const double cR = sqrt(gamma * pR / rR);

    /* S3 */
    const double rbar = 0.5 * (rL + rR), cbar = 0.5 * (cL + cR);
    double pstar = 0.5 * (pL + pR) - 0.5 * (uR - uL) * rbar * cbar;
    if (pstar < 0.0) pstar = 0.0;

    /* Eq. 5 */
    const double g = (gamma + 1.0) / (2.0 * gamma);
    const double qL = sqrt(1.0 + g * (fmax(pstar / pL, 1.0) - 1.0));
    const double qR = sqrt(1.0 + g * (fmax(pstar / pR, 1.0) - 1.0));
    const double dsL = -cL * qL;
    const double dsR = cR * qR;
    const double sL = uL + dsL;
    const double sR = uR + dsR;

    /* Eq. 4 */
    const double sstar = ((pR - rR * uR * dsR) - (pL - rL * uL * dsL)) / (rL * dsL - rR * dsR);

    /* physical fluxes and conserved states on both sides (Eq. 2) */
    const double eL = pL / (gamma - 1.0) + 0.5 * rL * (uL * uL + vL * vL + wL * wL);
    const double eR = pR / (gamma - 1.0) + 0.5 * rR * (uR * uR + vR * vR + wR * wR);
    const double UL[5] = { rL, rL * uL, rL * vL, rL * wL, eL };
    const double UR[5] = { rR, rR * uR, rR * vR, rR * wR, eR };
    const double FL[5] = { rL * uL, rL * uL * uL + pL, rL * uL * vL, rL * uL * wL, (eL + pL) * uL };
    const double FR[5] = { rR * uR, rR * uR * uR + pR, rR * uR * vR, rR * uR * wR, (eR + pR) * uR };

    if (sL >= 0.0) { for (int m = 0; m < 5; m++) F[m] = FL[m]; return; }
    if (sstar >= 0.0) {
        const double r = dsL / (sL - sstar); /* the ratio first: exactly 1 when s_star = u_L */
        const double Us[5] = { rL * r, rL * r * sstar, rL * r * vL, rL * r * wL,
                               rL * r * (eL / rL + (sstar - uL) * (sstar + pL / (rL * dsL))) };
        for (int m = 0; m < 5; m++) F[m] = FL[m] + sL * (Us[m] - UL[m]);
        return;
    }
    if (sR > 0.0) {
        const double r = dsR / (sR - sstar);
        const double Us[5] = { rR * r, rR * r * sstar, rR * r * vR, rR * r * wR,
                               rR * r * (eR / rR + (sstar - uR) * (sstar + pR / (rR * dsR))) };
        for (int m = 0; m < 5; m++) F[m] = FR[m] + sR * (Us[m] - UR[m]);
        return;
    }
    for (int m = 0; m < 5; m++) F[m] = FR[m];
}

/* ------------------------------------------------------------------------- */
/* geometry helper: ghost-padded primitive array W[5][pz][py][px] */
typedef struct {
    int n[3];   /* interior extents nx, ny, nz */
    int g[3];   /* ghost layers per axis: NGH if active, else 0 */
    int p[3];   /* padded extents */
    long long cells; /* padded cell count */
} orc_geom;

static orc_geom make_geom(int nx, int ny, int nz)
{
    orc_geom G;
    G.n[0] = nx; G.n[1] = ny; G.n[2] = nz;
    for (int d = 0; d < 3; d++) { G.g[d] = (G.n[d] > 1) ? NGH : 0; G.p[d] = G.n[d] + 2 * G.g[d]; }
    G.cells = (long long)G.p[0] * G.p[1] * G.p[2];
    return G;
}

/* index of padded cell with *interior-relative* coordinates (i,j,k), i in [-g, n+g) */
static inline long long pidx(const orc_geom *G, int i, int j, int k)
{
    return ((long long)(k + G->g[2]) * G->p[1] + (j + G->g[1])) * G->p[0] + (i + G->g[0]);
}

/* ------------------------------------------------------------------------- */
/* Sec. 3.1.1: ghost-zone fill on PRIMITIVES, faces only (S11).
 * The rules are printed for the left-x boundary, cells -i-1/2 (ghost) from +1/2 or
 * +i+1/2 (interior), 0 <= i <= n_gh-1, with v_x the INWARD normal component:
 *   Free:       q(-i-1/2) = q(1/2)
 *   Outflow:    Free, but v_x(-i-1/2) = min(v_x(1/2), 0)
 *   Reflecting: q(-i-1/2) = q(i+1/2), but v_x(-i-1/2) = -v_x(i+1/2)
 * Periodic edges are communication boundaries filled by direct copy.
 * For a high-side face the inward normal is -axis, so "min(v_in,0)" on the inward
 * component becomes max(v_axis, 0) on the axis component.
 * W is the padded array; axis d in {0,1,2}; applied for interior transverse coords. */
void orc_fill_ghosts_axis(double *W, int nx, int ny, int nz, int d, int bc_lo, int bc_hi)
{
    orc_geom G = make_geom(nx, ny, nz);
    if (G.g[d] == 0) return;
    const int n = G.n[d];
    const int d1 = (d + 1) % 3, d2 = (d + 2) % 3;
    const int ivn = IVX + d; /* slot of the velocity component normal to this face */
    for (int b = 0; b < G.n[d2]; b++)
        for (int a = 0; a < G.n[d1]; a++)
            for (int layer = 0; layer < NGH; layer++)
                for (int side = 0; side < 2; side++) {
                    const int bc = side ? bc_hi : bc_lo;
                    int ig, is; /* ghost and source coordinate along d */
                    if (side == 0) {
                        ig = -1 - layer;
                        if (bc == BC_PERIODIC) is = n - 1 - layer;
                        else if (bc == BC_REFLECT) is = layer;
                        else is = 0;
                    } else {
                        ig = n + layer;
                        if (bc == BC_PERIODIC) is = layer;
                        else if (bc == BC_REFLECT) is = n - 1 - layer;
                        else is = n - 1;
                    }
                    int cg[3], cs[3];
                    cg[d] = ig; cs[d] = is;
                    cg[d1] = cs[d1] = a;
                    cg[d2] = cs[d2] = b;
                    const long long jg = pidx(&G, cg[0], cg[1], cg[2]);
                    const long long js = pidx(&G, cs[0], cs[1], cs[2]);
                    for (int m = 0; m < 5; m++) W[m * G.cells + jg] = W[m * G.cells + js];
                    if (bc == BC_REFLECT) {
                        W[ivn * G.cells + jg] = -W[ivn * G.cells + js];
                    } else if (bc == BC_OUTFLOW) {
                        const double vn = W[ivn * G.cells + js];
                        /* inward component: +vn on the low side, -vn on the high side */
                        if (side == 0) W[ivn * G.cells + jg] = fmin(vn, 0.0);
                        else           W[ivn * G.cells + jg] = fmax(vn, 0.0);
                    }
                }
}

/* ------------------------------------------------------------------------- */
/* L(U) = - sum_d (F_{d,i+1/2} - F_{d,i-1/2}) / dx_d  on interior cells
 * (Fig. 3 green + magenta steps; Sec. 3.1-3.2).
 *   1. primitives on the interior
 *   2. ghost fill on primitives
 *   3. per active axis: PLM with minmod slopes, Delta x in the denominator
 *      (Eq. 3), then HLLC at every face.
 * Lout has the layout of U.  Returns 0, or -2 if allocation fails. */
/* order = 2: slope-limited PLM (Eq. 3); order = 1: piecewise-constant states (all slopes 0), used by the
 * predictor of the van Leer integrator (reading S15). */
static int flux_divergence_order(const double *U, int nx, int ny, int nz, double gamma, const int bc[6],
                                 double dx, double dy, double dz, double *Lout, long long *floor_hits, int order)
{
    orc_geom G = make_geom(nx, ny, nz);
    const long long N = (long long)nx * ny * nz;
    const double h[3] = { dx, dy, dz };
    double *W = (double *)malloc(sizeof(double) * 5 * G.cells);
    if (!W) return -2;
    memset(W, 0, sizeof(double) * 5 * G.cells);
    long long hits = 0;

    /* 1. primitive recovery */
#pragma omp parallel for reduction(+ : hits)
    for (int k = 0; k < nz; k++)
        for (int j = 0; j < ny; j++)
            for (int i = 0; i < nx; i++) {
                const long long c = ((long long)k * ny + j) * nx + i;
                double u[5], w[5];
                for (int m = 0; m < 5; m++) u[m] = U[m * N + c];
                orc_cons_to_prim(u, gamma, w, &hits);
                const long long q = pidx(&G, i, j, k);
                for (int m = 0; m < 5; m++) W[m * G.cells + q] = w[m];
            }
    if (floor_hits) *floor_hits += hits;

    /* 2. ghost zones */
    for (int d = 0; d < 3; d++) orc_fill_ghosts_axis(W, nx, ny, nz, d, bc[2 * d], bc[2 * d + 1]);

    for (long long c = 0; c < 5 * N; c++) Lout[c] = 0.0;

    /* 3. sweeps */
    for (int d = 0; d < 3; d++) {
        if (G.g[d] == 0) continue;
        const int n = G.n[d];
        const int d1 = (d + 1) % 3, d2 = (d + 2) % 3;
        /* normal-frame slots: u = v_d, v = v_{d1}, w = v_{d2} */
        const int su = IVX + d, sv = IVX + d1, sw = IVX + d2;
#pragma omp parallel for collapse(2)
        for (int b = 0; b < G.n[d2]; b++) {
            for (int a = 0; a < G.n[d1]; a++) {
                /* line buffers, index l = i + NGH for i in [-2, n+2) */
                double *q = (double *)malloc(sizeof(double) * 5 * (n + 2 * NGH));
                double *sig = (double *)malloc(sizeof(double) * 5 * (n + 2 * NGH));
                double *Fl = (double *)malloc(sizeof(double) * 5 * (n + 1)); /* face i+1/2, i=-1..n-1 -> slot i+1 */
                for (int i = -NGH; i < n + NGH; i++) {
                    int cc[3];
                    cc[d] = i; cc[d1] = a; cc[d2] = b;
                    const long long p = pidx(&G, cc[0], cc[1], cc[2]);
                    double *ql = q + 5 * (i + NGH);
                    ql[0] = W[IR * G.cells + p];
                    ql[1] = W[IP * G.cells + p];
                    ql[2] = W[su * G.cells + p];
                    ql[3] = W[sv * G.cells + p];
                    ql[4] = W[sw * G.cells + p];
                }
                /* slopes for cells i = -1..n (Eq. 3; Delta x directly in the denominator) */
                for (int i = -1; i <= n; i++)
                    for (int m = 0; m < 5; m++) {
                        const double qm = q[5 * (i - 1 + NGH) + m], q0 = q[5 * (i + NGH) + m],
                                     qp = q[5 * (i + 1 + NGH) + m];
                        sig[5 * (i + NGH) + m] = (order == 1) ? 0.0 : orc_minmod((q0 - qm) / h[d], (qp - q0) / h[d]);
                    }
                /* faces i+1/2, i = -1..n-1 */
                for (int i = -1; i <= n - 1; i++) {
                    double WL[5], WR[5];
                    for (int m = 0; m < 5; m++) {
                        WL[m] = q[5 * (i + NGH) + m] + 0.5 * h[d] * sig[5 * (i + NGH) + m];
                        WR[m] = q[5 * (i + 1 + NGH) + m] - 0.5 * h[d] * sig[5 * (i + 1 + NGH) + m];
                    }
                    orc_hllc(WL, WR, gamma, Fl + 5 * (i + 1));
                }
                /* flux difference; rotate momentum components back to (x,y,z) */
                for (int i = 0; i < n; i++) {
                    int cc[3];
                    cc[d] = i; cc[d1] = a; cc[d2] = b;
                    const long long c = ((long long)cc[2] * ny + cc[1]) * nx + cc[0];
                    const double *Fm = Fl + 5 * i, *Fp = Fl + 5 * (i + 1);
                    Lout[0 * N + c] -= (Fp[0] - Fm[0]) / h[d];
                    Lout[(1 + d) * N + c] -= (Fp[1] - Fm[1]) / h[d];
                    Lout[(1 + d1) * N + c] -= (Fp[2] - Fm[2]) / h[d];
                    Lout[(1 + d2) * N + c] -= (Fp[3] - Fm[3]) / h[d];
                    Lout[4 * N + c] -= (Fp[4] - Fm[4]) / h[d];
                }
                free(q); free(sig); free(Fl);
            }
        }
    }
    free(W);
    return 0;
}

/* ------------------------------------------------------------------------- */
/* L(U) of Eq. 2 with the paper's default scheme: slope-limited PLM states (Eq. 3) and HLLC fluxes
 * (Eq. 4-5) at every face of every active axis, differenced over the cell.  Lout: 5*nx*ny*nz doubles. */
int orc_flux_divergence(const double *U, int nx, int ny, int nz, double gamma, const int bc[6],
                        double dx, double dy, double dz, double *Lout, long long *floor_hits)
{
    return flux_divergence_order(U, nx, ny, nz, gamma, bc, dx, dy, dz, Lout, floor_hits, 2);
}

/* Sec. 3.3: the "memory-optimized second order van Leer integrator", whose prediction
 * sub-step does not enter the final result directly.  The paper prints no formulas; reading S15:
 * the predictor-corrector of van Leer as used in finite-volume codes,
 *     U^{n+1/2} = U^n + (dt/2) L_1(U^n)        L_1: piecewise-constant states at the faces (first order)
 *     U^{n+1}   = U^n +  dt    L_2(U^{n+1/2})  L_2: slope-limited PLM + HLLC, as in the Heun stages
 * Same ghost rules, floors and CFL formula as the Heun path.  Conservative: U^n only ever receives flux
 * differences.  Parity with Kratos' own choice is UNPINNED. */
int orc_step_vl(double *U, int nx, int ny, int nz, double gamma, const int bc[6],
                double dx, double dy, double dz, double dt, long long *floor_hits)
{
    const long long N5 = 5LL * nx * ny * nz;
    double *L = (double *)malloc(sizeof(double) * N5);
    double *Uh = (double *)malloc(sizeof(double) * N5);
    if (!L || !Uh) { free(L); free(Uh); return -2; }
    int rc = flux_divergence_order(U, nx, ny, nz, gamma, bc, dx, dy, dz, L, floor_hits, 1);
    if (rc) { free(L); free(Uh); return rc; }
#pragma omp parallel for
    for (long long c = 0; c < N5; c++) Uh[c] = U[c] + 0.5 * dt * L[c];
    rc = flux_divergence_order(Uh, nx, ny, nz, gamma, bc, dx, dy, dz, L, floor_hits, 2);
    if (rc) { free(L); free(Uh); return rc; }
#pragma omp parallel for
    for (long long c = 0; c < N5; c++) U[c] = U[c] + dt * L[c];
    free(L); free(Uh);
    return 0;
}

/* Sec. 3.3: one Heun (RK2) step of length dt.
 *   U1 = U0 + dt L(U0);  U = 1/2 U0 + 1/2 (U1 + dt L(U1))     (predictor enters with weight 1/2)
 * U is updated in place. */
int orc_step(double *U, int nx, int ny, int nz, double gamma, const int bc[6],
             double dx, double dy, double dz, double dt, long long *floor_hits)
{
    const long long N5 = 5LL * nx * ny * nz;
    double *L = (double *)malloc(sizeof(double) * N5);
    double *U1 = (double *)malloc(sizeof(double) * N5);
    if (!L || !U1) { free(L); free(U1); return -2; }
    int rc = orc_flux_divergence(U, nx, ny, nz, gamma, bc, dx, dy, dz, L, floor_hits);
    if (rc) { free(L); free(U1); return rc; }
#pragma omp parallel for
    for (long long c = 0; c < N5; c++) U1[c] = U[c] + dt * L[c];
    rc = orc_flux_divergence(U1, nx, ny, nz, gamma, bc, dx, dy, dz, L, floor_hits);
    if (rc) { free(L); free(U1); return rc; }
#pragma omp parallel for
    for (long long c = 0; c < N5; c++) U[c] = 0.5 * U[c] + 0.5 * (U1[c] + dt * L[c]);
    free(L); free(U1);
    return 0;
}

/* ------------------------------------------------------------------------- */
/* Sec. 3.1: time step "based on the CFL conditions", evaluated during
 * the variable conversion.  Reading S1 (sum form):
 *   dt = cfl / max_cells sum_{active d} (|v_d| + c) / dx_d,   c = sqrt(gamma p / rho). */
double orc_cfl_dt(const double *U, int nx, int ny, int nz, double gamma,
                  double dx, double dy, double dz, double cfl, long long *floor_hits)
{
    const long long N = (long long)nx * ny * nz;
    const int act[3] = { nx > 1, ny > 1, nz > 1 };
    const double h[3] = { dx, dy, dz };
    double rate_max = 0.0;
    long long hits = 0;
#pragma omp parallel for reduction(max : rate_max) reduction(+ : hits)
    for (long long c = 0; c < N; c++) {
        double u[5], w[5];
        for (int m = 0; m < 5; m++) u[m] = U[m * N + c];
        orc_cons_to_prim(u, gamma, w, &hits);
        const double cs = sqrt(gamma * w[IP] / w[IR]);
        double rate = 0.0;
        for (int d = 0; d < 3; d++)
            if (act[d]) rate += (fabs(w[IVX + d]) + cs) / h[d];
        if (rate > rate_max) rate_max = rate;
    }
    if (floor_hits) *floor_hits += hits;
    return cfl / rate_max;
}

/* ------------------------------------------------------------------------- */
/* Driver: repeat { dt = cfl_dt; clip to t_end; step } for at most nsteps steps or
 * until t reaches t_end (t_end <= 0: no end time).  Returns steps taken, <0 on error. */
static int run_with(int integrator, double *U, int nx, int ny, int nz, double gamma, const int bc[6],
                    double dx, double dy, double dz, double cfl, int nsteps, double t_end,
                    double *t_inout, long long *floor_hits)
{
    double t = *t_inout;
    int s = 0;
    for (; s < nsteps; s++) {
        if (t_end > 0.0 && t >= t_end) break;
        double dt = orc_cfl_dt(U, nx, ny, nz, gamma, dx, dy, dz, cfl, floor_hits);
        if (t_end > 0.0 && t + dt > t_end) dt = t_end - t;
        int rc = integrator ? orc_step_vl(U, nx, ny, nz, gamma, bc, dx, dy, dz, dt, floor_hits)
                            : orc_step(U, nx, ny, nz, gamma, bc, dx, dy, dz, dt, floor_hits);
        if (rc) return rc;
        t += dt;
    }
    *t_inout = t;
    return s;
}

int orc_run(double *U, int nx, int ny, int nz, double gamma, const int bc[6],
            double dx, double dy, double dz, double cfl, int nsteps, double t_end,
            double *t_inout, long long *floor_hits)
{
    return run_with(0, U, nx, ny, nz, gamma, bc, dx, dy, dz, cfl, nsteps, t_end, t_inout, floor_hits);
}

int orc_run_vl(double *U, int nx, int ny, int nz, double gamma, const int bc[6],
               double dx, double dy, double dz, double cfl, int nsteps, double t_end,
               double *t_inout, long long *floor_hits)
{
    return run_with(1, U, nx, ny, nz, gamma, bc, dx, dy, dz, cfl, nsteps, t_end, t_inout, floor_hits);
}

/* ------------------------------------------------------------------------- */
/* Sum of each conserved field over the interior, Neumaier-compensated (a plain fp64
 * sum over 10^8 cells would itself err at the 1e-13 level the conservation pin asks for). */
void orc_totals(const double *U, long long ncell, double out[5])
{
    for (int m = 0; m < 5; m++) {
        double s = 0.0, comp = 0.0;
        const double *f = U + m * ncell;
        for (long long c = 0; c < ncell; c++) {
            const double x = f[c];
            const double t = s + x;
            if (fabs(s) >= fabs(x)) comp += (s - t) + x;
            else comp += (x - t) + s;
            s = t;
        }
        out[m] = s + comp;
    }
}

/* threads the OpenMP loops will use (for bench.py's "cores" field) */
#ifdef _OPENMP
#include <omp.h>
int orc_num_threads(void) { return omp_get_max_threads(); }
#else
int orc_num_threads(void) { return 1; }
#endif
