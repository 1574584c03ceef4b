/*
 * hydro_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU oracle of GAMER-2's batched per-patch-group hydrodynamic solver
 * (arXiv 1712.07070).  It exists so that tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py can check and time the CUDA path against
 * something written independently from the paper.  Nothing under paper_1712_07070_b200/
 * imports, links or executes this file, and this file shares no code, header, table or helper
 * with the CUDA tree.
 *
 * What it follows (PAPER.md = /root/reference/PAPER.md, section 2.2 unless noted):
 *   - Euler equations, ideal gas, conserved (rho, mom, E); definitions of P, E_kin, E_the: L100
 *   - MHM (MUSCL-Hancock) and CTU ("6 Riemann solvers per cell per time-step"): L90
 *   - VL ("a variant of the MUSCL-Hancock scheme (VL; Falle 1991; van Leer 2006)", L90; Eq. (2) applies to it, L168):
 *     the half-step predictor is a first-order Godunov update of the cell averages (reading R26 of DESIGN.md)
 *   - PLM / PPM reconstruction on primitive variables, slope limiters: L94
 *   - Roe / HLLC / HLLE Riemann solvers: L94
 *   - dual-energy formalism with entropy s = P/rho^(gamma-1) and switch xi: L100
 *   - remedies (i) Roe -> HLLE on failed faces, (ii) first-order unsplit recompute: L104-105
 *   - boundary fluxes for the flux fix-up: L112
 *   - CFL conditions Eq. (1) (CTU) and Eq. (2) (MHM): L158-168
 *   - patch group = 16^3 cells (L242), 3 ghost zones (L300)
 * The paper defers every formula to the literature it names ("which we do not repeat here",
 * L92); the formulas below are the textbook ones (Toro 2009; Colella & Woodward 1984;
 * Colella 1990 / Stone et al. 2008; Roe 1981; Einfeldt et al. 1991) in the readings that
 * DESIGN.md section "Readings" lists one by one (R1..R20).
 *
 * Style: one patch group at a time, full-size intermediate arrays, nested loops in the order
 * the steps are stated, no tiling, no fusion.  OpenMP only over patch groups (the paper's own
 * CPU parallelisation, L258).  Build: gcc -O2 -ffp-contract=off -fopenmp (see oracle/build.py).
 *
 * Layouts (x fastest):  in [n_groups][NV][22][22][22],  out [n_groups][NV][16][16][16],
 * flux_out [n_groups][3 axes][3 planes][NV][16][16]  (plane p of axis d is the face at cell-face
 * index 8p of that axis; the two 16-long dims are the remaining axes in z,y,x order, slowest
 * first), group_speed [n_groups].  NV = 5 + n_scalar.
 *
 * Pins (tests/test_oracle_*.py): exact Riemann solution of Sod's tube, closed-form fluxes,
 * Roe identities, conservation on a periodic box, uniform-state invariance, x/y/z permutation
 * and mirror symmetry, 1-D reduction, exact reproduction of linear / parabolic data, single-wave
 * characteristic tracing, ghost-footprint, dual-energy / floor closed forms, CFL closed forms;
 * CTU transverse correction: 3-D contact advection against the 6-solve scheme written out, cells
 * rebuilt from the pinned building blocks, second-order diagonal advection; PPM overshoot branches:
 * hand-computed cases (both copies); characteristic limiting: R . limiter(L dW) with eigenvectors
 * written out from the literature; VL scheme: contact-advection closed form, cell rebuilt from
 * single-face solves; passive scalars: per-species conservation, bitwise independence, closed-form
 * renormalisation (DESIGN.md section 2 lists which test kills which mutation).
 * Parity unpinned: none of the functions exported here (the hybrid limiter and remedy (iii) are
 * not implemented at all).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define PS   16              /* cells per patch-group edge (L242)            */
#define NG   3               /* ghost cells per side (L300)                   */
#define NP   (PS + 2 * NG)   /* padded edge = 22                              */
#define NPC  (NP * NP * NP)  /* padded cells per group = 10648                */
#define NSMAX 8             /* passive scalars carried at most (L96 "an arbitrary number"; a compile-time bound here) */
#define NVMAX (5 + NSMAX)
#define IDX(i, j, k) ((((k) * NP) + (j)) * NP + (i))

enum { SCHEME_MHM = 1, SCHEME_CTU = 2, SCHEME_VL = 3 };
enum { RECON_PLM = 1, RECON_PPM = 2 };
enum { RSOLVER_ROE = 1, RSOLVER_HLLC = 2, RSOLVER_HLLE = 3, RSOLVER_EXACT = 4 };
enum { LIMITER_GMINMOD = 1, LIMITER_VANLEER = 2, LIMITER_VANALBADA = 3 };

typedef struct {
    int    limiter;            /* LIMITER_*                                              */
    double theta;              /* generalized-minmod parameter                           */
    int    n_scalar;           /* 0..NSMAX passively advected scalars (L96); with dual_energy the LAST one is the entropy (L100) */
    int    dual_energy;        /* 0/1                                                    */
    double de_xi;              /* switch E_the/E_kin < xi (L100)                         */
    double min_dens, min_pres, min_temp;   /* floors; 0 = off                            */
    int    remedy_first_order; /* remedy (ii), L105                                      */
    int    char_limiting;      /* 0: slopes limited in primitive variables; 1: in characteristic ones (L94) */
    int    renormalize;        /* 1: after the update rescale the passive scalars (not the entropy) so that they sum to rho (L96) */
} orc_opts;

typedef struct {
    int64_t n_riemann;        /* Riemann solver calls (all passes, incl. halo faces)     */
    int64_t n_riemann_final;  /* calls of the final pass (faces bounding interior cells) */
    int64_t n_roe_fallback;   /* remedy (i) taken                                        */
    int64_t n_pred_revert;    /* predictor / tracing / correction states reverted        */
    int64_t n_first_order;    /* remedy (ii) taken                                       */
    int64_t n_dual_fix;       /* cells whose E was rebuilt from the entropy              */
    int64_t n_floor;          /* cells touched by a floor in the closing step            */
    int64_t n_unphysical;     /* cells still unphysical at the end                       */
} orc_stats;

typedef struct {
    double gamma, gm1;
    int    nv;
    orc_opts o;
} ctx_t;

/* ------------------------------------------------------------------------------------------
 * O1: conserved <-> primitive (E_the = E_tot - E_kin, P from the ideal gas law)
 * U = (rho, mx, my, mz, E [, s]);  W = (rho, vx, vy, vz, P [, q = s/rho])
 * ---------------------------------------------------------------------------------------- */
static void cons2prim(const ctx_t *c, const double *U, double *W)
{
    double rho = U[0];
    W[0] = rho;
    W[1] = U[1] / rho;
    W[2] = U[2] / rho;
    W[3] = U[3] / rho;
    double ekin = 0.5 * (U[1] * U[1] + U[2] * U[2] + U[3] * U[3]) / rho;
    W[4] = c->gm1 * (U[4] - ekin);
    for (int v = 5; v < c->nv; ++v) W[v] = U[v] / rho;   /* q_k = s_k / rho */
}

static void prim2cons(const ctx_t *c, const double *W, double *U)
{
    double rho = W[0];
    U[0] = rho;
    U[1] = rho * W[1];
    U[2] = rho * W[2];
    U[3] = rho * W[3];
    U[4] = W[4] / c->gm1 + 0.5 * rho * (W[1] * W[1] + W[2] * W[2] + W[3] * W[3]);
    for (int v = 5; v < c->nv; ++v) U[v] = rho * W[v];
}

static int floors_set(const ctx_t *c)
{
    return c->o.min_dens > 0.0 || c->o.min_pres > 0.0 || c->o.min_temp > 0.0;
}

/* floors on a primitive state (reading R14): rho >= min_dens, P >= max(min_pres, rho*min_temp) */
static void floor_prim(const ctx_t *c, double *W)
{
    if (c->o.min_dens > 0.0 && W[0] < c->o.min_dens) W[0] = c->o.min_dens;
    double pf = c->o.min_pres;
    double pt = W[0] * c->o.min_temp;
    if (pt > pf) pf = pt;
    if (pf > 0.0 && W[4] < pf) W[4] = pf;
}

/* physical flux along axis d (0,1,2) of the state given both as W and as U */
static void phys_flux(const ctx_t *c, int d, const double *W, const double *U, double *F)
{
    double vn = W[1 + d];
    F[0] = U[0] * vn;
    F[1] = U[1] * vn;
    F[2] = U[2] * vn;
    F[3] = U[3] * vn;
    F[1 + d] += W[4];
    F[4] = vn * (U[4] + W[4]);
    for (int v = 5; v < c->nv; ++v) F[v] = U[v] * vn;
}

/* ------------------------------------------------------------------------------------------
 * O2: limited slope (L94: "generalized minmod limiter, van Leer-type limiter, van Albada-type")
 * ---------------------------------------------------------------------------------------- */
static double limited_slope(const ctx_t *c, double dL, double dR)
{
    if (dL * dR <= 0.0) return 0.0;
    switch (c->o.limiter) {
    case LIMITER_VANLEER:
        return 2.0 * dL * dR / (dL + dR);
    case LIMITER_VANALBADA:
        return dL * dR * (dL + dR) / (dL * dL + dR * dR);
    default: {
        double th = c->o.theta;
        double a = th * fabs(dL), b = 0.5 * fabs(dL + dR), e = th * fabs(dR);
        double m = a < b ? a : b;
        if (e < m) m = e;
        return dR > 0.0 ? m : -m;
    }
    }
}

/* ------------------------------------------------------------------------------------------
 * O3: face values of one cell along one axis from the five cell values w[-2..2] of one
 * primitive variable.  Returns wm (at face i-1/2) and wp (at face i+1/2).
 * PLM (van Leer 1979): W -/+ slope/2.   PPM (Colella & Woodward 1984): fourth-order interface
 * values from limited slopes, then monotonisation; no steepening, no flattening (R5).
 * ---------------------------------------------------------------------------------------- */
static void face_values(const ctx_t *c, int recon, const double w[5], double *wm, double *wp)
{
    const double *q = w + 2; /* q[-2..2] */
    if (recon == RECON_PLM) {
        double s = limited_slope(c, q[0] - q[-1], q[1] - q[0]);
        *wm = q[0] - 0.5 * s;
        *wp = q[0] + 0.5 * s;
        return;
    }
    double sm = limited_slope(c, q[-1] - q[-2], q[0] - q[-1]);
    double s0 = limited_slope(c, q[0] - q[-1], q[1] - q[0]);
    double sp = limited_slope(c, q[1] - q[0], q[2] - q[1]);
    double m = 0.5 * (q[-1] + q[0]) - (s0 - sm) / 6.0;
    double p = 0.5 * (q[0] + q[1]) - (sp - s0) / 6.0;
    if ((p - q[0]) * (q[0] - m) <= 0.0) {
        m = q[0];
        p = q[0];
    } else {
        double D = p - m;
        double C = q[0] - 0.5 * (m + p);
        if (D * C > D * D / 6.0)
            m = 3.0 * q[0] - 2.0 * p;
        else if (D * C < -D * D / 6.0)
            p = 3.0 * q[0] - 2.0 * m;
    }
    *wm = m;
    *wp = p;
}

/* ------------------------------------------------------------------------------------------
 * O5: Riemann solvers on x-normal states.  UL, UR conserved (rho, mn, mt1, mt2, E [, s]).
 * ---------------------------------------------------------------------------------------- */
typedef struct {
    double rho, u, v, w, P, E, c, H;
} rstate_t;

static void rstate(const ctx_t *c, const double *U, rstate_t *s)
{
    s->rho = U[0];
    s->u = U[1] / U[0];
    s->v = U[2] / U[0];
    s->w = U[3] / U[0];
    s->E = U[4];
    s->P = c->gm1 * (U[4] - 0.5 * (U[1] * U[1] + U[2] * U[2] + U[3] * U[3]) / U[0]);
    s->c = sqrt(c->gamma * s->P / s->rho);
    s->H = (s->E + s->P) / s->rho;
}

static void xflux(const rstate_t *s, const double *U, double *F)
{
    F[0] = U[1];
    F[1] = U[1] * s->u + s->P;
    F[2] = U[2] * s->u;
    F[3] = U[3] * s->u;
    F[4] = s->u * (s->E + s->P);
}

typedef struct {
    double u, v, w, H, q2, a2, a;
} roeavg_t;

static void roe_average(const ctx_t *c, const rstate_t *L, const rstate_t *R, roeavg_t *r)
{
    double wl = sqrt(L->rho), wr = sqrt(R->rho), den = wl + wr;
    r->u = (wl * L->u + wr * R->u) / den;
    r->v = (wl * L->v + wr * R->v) / den;
    r->w = (wl * L->w + wr * R->w) / den;
    r->H = (wl * L->H + wr * R->H) / den;
    r->q2 = r->u * r->u + r->v * r->v + r->w * r->w;
    r->a2 = c->gm1 * (r->H - 0.5 * r->q2);
    r->a = r->a2 > 0.0 ? sqrt(r->a2) : 0.0;
}

/* HLLE (Einfeldt et al. 1991) */
static void solve_hlle(const rstate_t *L, const rstate_t *R, const roeavg_t *r, const double *UL,
                       const double *UR, double *F)
{
    double FL[5], FR[5];
    xflux(L, UL, FL);
    xflux(R, UR, FR);
    double bl = fmin(r->u - r->a, L->u - L->c);
    double br = fmax(r->u + r->a, R->u + R->c);
    double bm = fmin(bl, 0.0), bp = fmax(br, 0.0);
    for (int v = 0; v < 5; ++v)
        F[v] = (bp * FL[v] - bm * FR[v] + bp * bm * (UR[v] - UL[v])) / (bp - bm);
}

/* HLLC (Toro 2009, ch. 10) with Einfeldt wave-speed bounds (R11) */
static void solve_hllc(const rstate_t *L, const rstate_t *R, const roeavg_t *r, const double *UL,
                       const double *UR, double *F)
{
    double FL[5], FR[5];
    xflux(L, UL, FL);
    xflux(R, UR, FR);
    double SL = fmin(r->u - r->a, L->u - L->c);
    double SR = fmax(r->u + r->a, R->u + R->c);
    if (SL >= 0.0) {
        for (int v = 0; v < 5; ++v) F[v] = FL[v];
        return;
    }
    if (SR <= 0.0) {
        for (int v = 0; v < 5; ++v) F[v] = FR[v];
        return;
    }
    double ml = L->rho * (SL - L->u), mr = R->rho * (SR - R->u);
    double SS = (R->P - L->P + L->u * ml - R->u * mr) / (ml - mr);
    const rstate_t *K;
    const double *UK, *FK;
    double SK;
    if (SS >= 0.0) {
        K = L, UK = UL, FK = FL, SK = SL;
    } else {
        K = R, UK = UR, FK = FR, SK = SR;
    }
    double fac = K->rho * (SK - K->u) / (SK - SS);
    double Us[5];
    Us[0] = fac;
    Us[1] = fac * SS;
    Us[2] = fac * K->v;
    Us[3] = fac * K->w;
    Us[4] = fac * (K->E / K->rho + (SS - K->u) * (SS + K->P / (K->rho * (SK - K->u))));
    for (int v = 0; v < 5; ++v) F[v] = FK[v] + SK * (Us[v] - UK[v]);
}

/* Roe (Roe 1981; Toro 2009 sect. 11.2.2/11.3), no entropy fix (R9).
 * Returns 1 if an intermediate state is unphysical (remedy (i) must be taken), else 0. */
static int solve_roe(const ctx_t *c, const rstate_t *L, const rstate_t *R, const roeavg_t *r,
                     const double *UL, const double *UR, double *F)
{
    if (!(r->a2 > 0.0)) return 1;
    double FL[5], FR[5], dU[5];
    xflux(L, UL, FL);
    xflux(R, UR, FR);
    for (int v = 0; v < 5; ++v) dU[v] = UR[v] - UL[v];
    double u = r->u, vv = r->v, w = r->w, H = r->H, a = r->a;
    double a3 = dU[2] - vv * dU[0];
    double a4 = dU[3] - w * dU[0];
    double d5 = dU[4] - a3 * vv - a4 * w;
    double a2 = c->gm1 / r->a2 * (dU[0] * (H - u * u) + u * dU[1] - d5);
    double a1 = (dU[0] * (u + a) - dU[1] - a * a2) / (2.0 * a);
    double a5 = dU[0] - (a1 + a2);
    double K1[5] = {1.0, u - a, vv, w, H - u * a};
    double K2[5] = {1.0, u, vv, w, 0.5 * r->q2};
    double K3[5] = {0.0, 0.0, 1.0, 0.0, vv};
    double K4[5] = {0.0, 0.0, 0.0, 1.0, w};
    double K5[5] = {1.0, u + a, vv, w, H + u * a};
    /* remedy (i), L104: intermediate states U_L + a1 K1 and U_R - a5 K5 */
    double Ua[5], Ub[5];
    for (int v = 0; v < 5; ++v) {
        Ua[v] = UL[v] + a1 * K1[v];
        Ub[v] = UR[v] - a5 * K5[v];
    }
    double Pa = c->gm1 * (Ua[4] - 0.5 * (Ua[1] * Ua[1] + Ua[2] * Ua[2] + Ua[3] * Ua[3]) / Ua[0]);
    double Pb = c->gm1 * (Ub[4] - 0.5 * (Ub[1] * Ub[1] + Ub[2] * Ub[2] + Ub[3] * Ub[3]) / Ub[0]);
    if (!(Ua[0] > 0.0) || !(Ub[0] > 0.0) || !(Pa > 0.0) || !(Pb > 0.0)) return 1;
    double l1 = fabs(u - a), l2 = fabs(u), l5 = fabs(u + a);
    for (int v = 0; v < 5; ++v)
        F[v] = 0.5 * (FL[v] + FR[v]) -
               0.5 * (l1 * a1 * K1[v] + l2 * (a2 * K2[v] + a3 * K3[v] + a4 * K4[v]) + l5 * a5 * K5[v]);
    return 0;
}

/* Exact Riemann solver ("exact solver based on Toro (2009)"; Toro ch. 4), reading R21 of DESIGN.md:
 *  - pressure function f_K(p) of Toro eqs. 4.6-4.7 (shock branch for p > p_K, rarefaction branch otherwise) and its
 *    derivative (eq. 4.37), star pressure from Newton-Raphson on f_L + f_R + (u_R - u_L) = 0 (eq. 4.5);
 *  - first guess: the two-rarefaction value p_TR (eq. 4.46), exact when both waves are rarefactions and always
 *    positive; if its numerator is not positive the data generate vacuum (eq. 4.40) and the solver reports failure
 *    (the caller falls back to HLLE, as for remedy (i));
 *  - iterate until 2|p_new - p_old| / (p_new + p_old) < 1e-6 (Toro's TOL), then ONE more step, at most 30 steps;
 *    a negative iterate is reset to 1e-6 of the guess;
 *  - u* from eq. 4.9, state at x/t = 0 sampled as in Toro section 4.5, transverse velocities taken from the side
 *    of the contact the axis lies on (u* >= 0: left), flux = physical flux of that state. */
static void pressure_fn(double p, double rho, double pk, double ck, double gamma, double *f, double *df)
{
    if (p > pk) {
        double A = 2.0 / ((gamma + 1.0) * rho), B = (gamma - 1.0) / (gamma + 1.0) * pk;
        double q = sqrt(A / (p + B));
        *f = (p - pk) * q;
        *df = q * (1.0 - 0.5 * (p - pk) / (B + p));
    } else {
        double pr = p / pk;
        *f = 2.0 * ck / (gamma - 1.0) * (pow(pr, (gamma - 1.0) / (2.0 * gamma)) - 1.0);
        *df = pow(pr, -(gamma + 1.0) / (2.0 * gamma)) / (rho * ck);
    }
}

static int solve_exact(const ctx_t *c, const rstate_t *L, const rstate_t *R, double *F)
{
    const double g = c->gamma, gm1 = g - 1.0, gp1 = g + 1.0, z = gm1 / (2.0 * g);
    const double du = R->u - L->u;
    const double num = L->c + R->c - 0.5 * gm1 * du;
    if (!(num > 0.0)) return 1;                                   /* vacuum is generated */
    const double p0 = pow(num / (L->c / pow(L->P, z) + R->c / pow(R->P, z)), 1.0 / z);
    double p = p0, fl, dfl, fr, dfr;
    int extra = 0;
    for (int it = 0; it < 30; ++it) {
        pressure_fn(p, L->rho, L->P, L->c, g, &fl, &dfl);
        pressure_fn(p, R->rho, R->P, R->c, g, &fr, &dfr);
        double pn = p - (fl + fr + du) / (dfl + dfr);
        if (!(pn > 0.0)) pn = 1e-6 * p0;
        const double change = 2.0 * fabs(pn - p) / (pn + p);
        p = pn;
        if (extra) break;
        if (change < 1e-6) extra = 1;
    }
    pressure_fn(p, L->rho, L->P, L->c, g, &fl, &dfl);
    pressure_fn(p, R->rho, R->P, R->c, g, &fr, &dfr);
    const double us = 0.5 * (L->u + R->u) + 0.5 * (fr - fl);
    double rho, u, P;
    const rstate_t *K = us >= 0.0 ? L : R;
    if (us >= 0.0) {                                              /* x/t = 0 lies left of the contact */
        if (p > L->P) {                                           /* left shock */
            double sl = L->u - L->c * sqrt(gp1 / (2.0 * g) * p / L->P + gm1 / (2.0 * g));
            if (0.0 <= sl) { rho = L->rho; u = L->u; P = L->P; }
            else { rho = L->rho * ((p / L->P + gm1 / gp1) / (gm1 / gp1 * p / L->P + 1.0)); u = us; P = p; }
        } else {                                                  /* left rarefaction */
            double shl = L->u - L->c, stl = us - L->c * pow(p / L->P, z);
            if (0.0 <= shl) { rho = L->rho; u = L->u; P = L->P; }
            else if (0.0 >= stl) { rho = L->rho * pow(p / L->P, 1.0 / g); u = us; P = p; }
            else {
                double cf = 2.0 / gp1 + gm1 / (gp1 * L->c) * L->u;
                rho = L->rho * pow(cf, 2.0 / gm1);
                u = 2.0 / gp1 * (L->c + 0.5 * gm1 * L->u);
                P = L->P * pow(cf, 2.0 * g / gm1);
            }
        }
    } else {
        if (p > R->P) {                                           /* right shock */
            double sr = R->u + R->c * sqrt(gp1 / (2.0 * g) * p / R->P + gm1 / (2.0 * g));
            if (0.0 >= sr) { rho = R->rho; u = R->u; P = R->P; }
            else { rho = R->rho * ((p / R->P + gm1 / gp1) / (gm1 / gp1 * p / R->P + 1.0)); u = us; P = p; }
        } else {                                                  /* right rarefaction */
            double shr = R->u + R->c, str_ = us + R->c * pow(p / R->P, z);
            if (0.0 >= shr) { rho = R->rho; u = R->u; P = R->P; }
            else if (0.0 <= str_) { rho = R->rho * pow(p / R->P, 1.0 / g); u = us; P = p; }
            else {
                double cf = 2.0 / gp1 - gm1 / (gp1 * R->c) * R->u;
                rho = R->rho * pow(cf, 2.0 / gm1);
                u = 2.0 / gp1 * (-R->c + 0.5 * gm1 * R->u);
                P = R->P * pow(cf, 2.0 * g / gm1);
            }
        }
    }
    const double E = P / gm1 + 0.5 * rho * (u * u + K->v * K->v + K->w * K->w);
    F[0] = rho * u;
    F[1] = rho * u * u + P;
    F[2] = rho * u * K->v;
    F[3] = rho * u * K->w;
    F[4] = u * (E + P);
    return 0;
}

/* flux through a face normal to axis d;  UL/UR full conserved states in x,y,z order */
static void riemann(const ctx_t *c, int solver, int d, const double *UL, const double *UR, double *F,
                    orc_stats *st)
{
    int n = 1 + d, t1 = 1 + (d + 1) % 3, t2 = 1 + (d + 2) % 3;
    double ul[5] = {UL[0], UL[n], UL[t1], UL[t2], UL[4]};
    double ur[5] = {UR[0], UR[n], UR[t1], UR[t2], UR[4]};
    double f[5];
    rstate_t L, R;
    roeavg_t r;
    rstate(c, ul, &L);
    rstate(c, ur, &R);
    roe_average(c, &L, &R, &r);
    st->n_riemann++;
    if (solver == RSOLVER_ROE) {
        if (solve_roe(c, &L, &R, &r, ul, ur, f)) {
            st->n_roe_fallback++;
            solve_hlle(&L, &R, &r, ul, ur, f); /* R10: HLLE is the fallback */
        }
    } else if (solver == RSOLVER_HLLC) {
        solve_hllc(&L, &R, &r, ul, ur, f);
    } else if (solver == RSOLVER_EXACT) {
        if (solve_exact(c, &L, &R, f)) {
            st->n_roe_fallback++;
            solve_hlle(&L, &R, &r, ul, ur, f); /* R21: vacuum-generating data fall back to HLLE */
        }
    } else {
        solve_hlle(&L, &R, &r, ul, ur, f);
    }
    F[0] = f[0];
    F[n] = f[1];
    F[t1] = f[2];
    F[t2] = f[3];
    F[4] = f[4];
    for (int v = 5; v < c->nv; ++v) { /* R12: every passive scalar rides the mass flux, upwinded */
        double ql = UL[v] / UL[0], qr = UR[v] / UR[0];
        F[v] = f[0] >= 0.0 ? f[0] * ql : f[0] * qr;
    }
}

/* ------------------------------------------------------------------------------------------
 * O4-CTU(a): characteristic tracing over dt/2 of one cell along one axis (Colella 1990;
 * Stone et al. 2008 sect. 4.2).  W: cell-centred primitive (rho, vn, vt1, vt2, P [, q]) with the
 * traced axis rotated to "n"; wm/wp: untraced face values; chi = dt/dh.  Output tm/tp.
 * Only waves moving toward the face are summed (R7).
 * ---------------------------------------------------------------------------------------- */
static void project(const double *dW, double rho, double cs, int nv, double *amp)
{
    double c2 = cs * cs;
    amp[0] = (dW[4] - rho * cs * dW[1]) / (2.0 * c2); /* v - c        */
    amp[1] = dW[0] - dW[4] / c2;                       /* entropy      */
    amp[2] = dW[2];                                    /* shear        */
    amp[3] = dW[3];                                    /* shear        */
    amp[4] = (dW[4] + rho * cs * dW[1]) / (2.0 * c2);  /* v + c        */
    for (int v = 5; v < nv; ++v) amp[v] = dW[v];       /* scalars      */
}

static void add_wave(double *T, int alpha, double amp, double rho, double cs)
{
    switch (alpha) {
    case 0: T[0] += amp; T[1] -= amp * cs / rho; T[4] += amp * cs * cs; break;
    case 1: T[0] += amp; break;
    case 2: T[2] += amp; break;
    case 3: T[3] += amp; break;
    case 4: T[0] += amp; T[1] += amp * cs / rho; T[4] += amp * cs * cs; break;
    default: T[alpha] += amp; break;   /* passive scalar alpha: its own characteristic field, speed vn */
    }
}

static void trace_cell(const ctx_t *c, int recon, const double *W, const double *wm, const double *wp,
                       double lam_r, double *tm, double *tp)
{
    int nv = c->nv;
    double rho = W[0], vn = W[1], cs = sqrt(c->gamma * W[4] / W[0]);
    double lam[NVMAX] = {vn - cs, vn, vn, vn, vn + cs};
    for (int a = 5; a < nv; ++a) lam[a] = vn;
    double chi[NVMAX];
    for (int a = 0; a < nv; ++a) chi[a] = lam[a] * lam_r;
    double chi5p = chi[4] > 0.0 ? chi[4] : 0.0;
    double chi1m = chi[0] < 0.0 ? chi[0] : 0.0;
    double d[NVMAX], w6[NVMAX], vec[NVMAX], amp[NVMAX];
    for (int v = 0; v < nv; ++v) {
        d[v] = wp[v] - wm[v];
        w6[v] = recon == RECON_PPM ? 6.0 * (W[v] - 0.5 * (wm[v] + wp[v])) : 0.0;
    }
    /* reference states: average over the domain of dependence of the fastest wave toward the face */
    for (int v = 0; v < nv; ++v) {
        tp[v] = wp[v] - 0.5 * chi5p * (d[v] - (1.0 - (2.0 / 3.0) * chi5p) * w6[v]);
        tm[v] = wm[v] - 0.5 * chi1m * (d[v] + (1.0 + (2.0 / 3.0) * chi1m) * w6[v]);
    }
    /* corrections for the slower waves that also reach the face */
    for (int a = 0; a < nv; ++a) {
        if (lam[a] > 0.0) {
            double A = 0.5 * (chi5p - chi[a]);
            double B = (chi5p * chi5p - chi[a] * chi[a]) / 3.0;
            for (int v = 0; v < nv; ++v) vec[v] = A * (d[v] - w6[v]) + B * w6[v];
            project(vec, rho, cs, nv, amp);
            add_wave(tp, a, amp[a], rho, cs);
        } else if (lam[a] < 0.0) {
            double C = 0.5 * (chi1m - chi[a]);
            double D = (chi1m * chi1m - chi[a] * chi[a]) / 3.0;
            for (int v = 0; v < nv; ++v) vec[v] = C * (d[v] + w6[v]) + D * w6[v];
            project(vec, rho, cs, nv, amp);
            add_wave(tm, a, amp[a], rho, cs);
        }
    }
}

/* ------------------------------------------------------------------------------------------
 * O7: closing step on one updated cell
 * ---------------------------------------------------------------------------------------- */
static int is_physical(const ctx_t *c, const double *U)
{
    for (int v = 0; v < c->nv; ++v)
        if (!isfinite(U[v])) return 0;
    if (!(U[0] > 0.0)) return 0;
    double P = c->gm1 * (U[4] - 0.5 * (U[1] * U[1] + U[2] * U[2] + U[3] * U[3]) / U[0]);
    return P > 0.0;
}

/* dual-energy formalism, L100 (R13): below the switch rebuild E from s, else resynchronise s */
static void dual_energy_fix(const ctx_t *c, double *U, orc_stats *st)
{
    if (!c->o.dual_energy || !(U[0] > 0.0)) return;
    double ekin = 0.5 * (U[1] * U[1] + U[2] * U[2] + U[3] * U[3]) / U[0];
    double ethe = U[4] - ekin;
    double rg = pow(U[0], c->gm1);
    if (ethe < c->o.de_xi * ekin) {
        double P = U[c->nv - 1] * rg;
        U[4] = ekin + P / c->gm1;
        st->n_dual_fix++;
    } else {
        U[c->nv - 1] = c->gm1 * ethe / rg;
    }
}

static void floor_cons(const ctx_t *c, double *U, orc_stats *st)
{
    int touched = 0;
    if (c->o.min_dens > 0.0 && U[0] < c->o.min_dens) {
        U[0] = c->o.min_dens;
        touched = 1;
    }
    double ekin = 0.5 * (U[1] * U[1] + U[2] * U[2] + U[3] * U[3]) / U[0];
    double P = c->gm1 * (U[4] - ekin);
    double pf = c->o.min_pres, pt = U[0] * c->o.min_temp;
    if (pt > pf) pf = pt;
    if (pf > 0.0 && P < pf) {
        U[4] = ekin + pf / c->gm1;
        if (c->o.dual_energy) U[c->nv - 1] = pf / pow(U[0], c->gm1);
        touched = 1;
    }
    st->n_floor += touched;
}

/* L96: "an arbitrary number of chemical species, which can be renormalized after every update to ensure that the sum
 * of their mass fractions equals unity": s_k <- s_k * rho / sum_k s_k over the passive scalars -- all of them, except the
 * last one when it is the entropy of the dual-energy formalism (reading R27).  A non-positive sum is left alone. */
static void renormalize_scalars(const ctx_t *c, double *U)
{
    if (!c->o.renormalize) return;
    int last = c->nv - (c->o.dual_energy ? 1 : 0);
    double sum = 0.0;
    for (int v = 5; v < last; ++v) sum = sum + U[v];
    if (!(sum > 0.0)) return;
    double f = U[0] / sum;
    for (int v = 5; v < last; ++v) U[v] = U[v] * f;
}

/* O9: CFL signal speed of one cell (Eq. 1 for CTU, Eq. 2 for MHM; L158-168) */
static double signal_speed(const ctx_t *c, int scheme, const double *U)
{
    double W[NVMAX];
    cons2prim(c, U, W);
    floor_prim(c, W);
    double cs = sqrt(c->gamma * W[4] / W[0]);
    double ax = fabs(W[1]), ay = fabs(W[2]), az = fabs(W[3]);
    if (scheme != SCHEME_CTU) return ax + ay + az + 3.0 * cs;   /* Eq. (2): MHM and VL (L168) */
    double m = ax > ay ? ax : ay;
    if (az > m) m = az;
    return m + cs;
}

/* ------------------------------------------------------------------------------------------
 * one patch group
 * ---------------------------------------------------------------------------------------- */
typedef struct {
    double *W;    /* [nv][NPC]           primitives                                  */
    double *FS;   /* [3][2][nv][NPC]     face states (conserved), s=0: minus, 1: plus */
    double *TS;   /* [3][2][nv][NPC]     CTU traced states (conserved)                */
    double *F1;   /* [3][nv][NPC]        CTU first-pass flux at face c + e_d/2        */
    double *FX;   /* [3][nv][NPC]        final flux at face c + e_d/2                 */
    double *WH;   /* [nv][NPC]           VL: primitives of the half-step state        */
} work_t;

#define FSI(d, s, v, n) ((((size_t)(d) * 2 + (s)) * nv + (v)) * NPC + (n))
#define FLI(d, v, n) (((size_t)(d) * nv + (v)) * NPC + (n))

static const int STEP[3] = {1, NP, NP * NP};

/* Limited slope vector of one cell in CHARACTERISTIC variables (L94 "applied to either primitive or characteristic
 * variables"; Stone et al. 2008 sect. 4.2.1, reading R22): the left and right differences of the rotated primitive
 * state are projected on the left eigenvectors evaluated at the cell itself (project), each characteristic amplitude
 * is limited by the same limiter as in the primitive case, and the limited amplitudes are multiplied back by the
 * right eigenvectors (add_wave).  Wl, Wc, Wr: rotated (rho, vn, vt1, vt2, P [, q]) of cells j-1, j, j+1. */
static void add_wave(double *T, int alpha, double amp, double rho, double cs);
static void project(const double *dW, double rho, double cs, int nv, double *amp);

static void char_slope(const ctx_t *c, const double *Wl, const double *Wc, const double *Wr, double *slope)
{
    int nv = c->nv;
    double dL[NVMAX], dR[NVMAX], aL[NVMAX], aR[NVMAX];
    double rho = Wc[0], cs = sqrt(c->gamma * Wc[4] / Wc[0]);
    for (int v = 0; v < nv; ++v) {
        dL[v] = Wc[v] - Wl[v];
        dR[v] = Wr[v] - Wc[v];
        slope[v] = 0.0;
    }
    project(dL, rho, cs, nv, aL);
    project(dR, rho, cs, nv, aR);
    for (int a = 0; a < nv; ++a) add_wave(slope, a, limited_slope(c, aL[a], aR[a]), rho, cs);
}

static void gather_face_values(const ctx_t *c, int recon, const double *W, int n, int d, double *wm,
                               double *wp)
{
    int nv = c->nv;
    if (c->o.char_limiting) {
        /* rotated copies of cells n-2 .. n+2 along d (PLM uses n-1 .. n+1 only) */
        int cn = 1 + d, c1 = 1 + (d + 1) % 3, c2 = 1 + (d + 2) % 3;
        int R = recon == RECON_PPM ? 2 : 1;
        double Wr[5][NVMAX], sl[3][NVMAX], rm[NVMAX], rp[NVMAX];
        for (int m = -R; m <= R; ++m) {
            const double *q = W + n + m * STEP[d];
            Wr[m + 2][0] = q[0];
            Wr[m + 2][1] = q[(size_t)cn * NPC];
            Wr[m + 2][2] = q[(size_t)c1 * NPC];
            Wr[m + 2][3] = q[(size_t)c2 * NPC];
            Wr[m + 2][4] = q[(size_t)4 * NPC];
            for (int v = 5; v < nv; ++v) Wr[m + 2][v] = q[(size_t)v * NPC];
        }
        if (recon == RECON_PLM) {
            char_slope(c, Wr[1], Wr[2], Wr[3], sl[1]);
            for (int v = 0; v < nv; ++v) {
                rm[v] = Wr[2][v] - 0.5 * sl[1][v];
                rp[v] = Wr[2][v] + 0.5 * sl[1][v];
            }
        } else {
            for (int j = 0; j < 3; ++j) char_slope(c, Wr[j], Wr[j + 1], Wr[j + 2], sl[j]);   /* cells n-1, n, n+1 */
            for (int v = 0; v < nv; ++v) {
                double q0 = Wr[2][v];
                double m = 0.5 * (Wr[1][v] + q0) - (sl[1][v] - sl[0][v]) / 6.0;
                double p = 0.5 * (q0 + Wr[3][v]) - (sl[2][v] - sl[1][v]) / 6.0;
                if ((p - q0) * (q0 - m) <= 0.0) {
                    m = q0;
                    p = q0;
                } else {
                    double D = p - m, C = q0 - 0.5 * (m + p);
                    if (D * C > D * D / 6.0) m = 3.0 * q0 - 2.0 * p;
                    else if (D * C < -D * D / 6.0) p = 3.0 * q0 - 2.0 * m;
                }
                rm[v] = m;
                rp[v] = p;
            }
        }
        /* back to the natural component order */
        wm[0] = rm[0]; wm[cn] = rm[1]; wm[c1] = rm[2]; wm[c2] = rm[3]; wm[4] = rm[4];
        wp[0] = rp[0]; wp[cn] = rp[1]; wp[c1] = rp[2]; wp[c2] = rp[3]; wp[4] = rp[4];
        for (int v = 5; v < nv; ++v) { wm[v] = rm[v]; wp[v] = rp[v]; }
        return;
    }
    for (int v = 0; v < nv; ++v) {
        double w[5];
        const double *q = W + (size_t)v * NPC + n;
        if (recon == RECON_PPM) {
            for (int m = -2; m <= 2; ++m) w[m + 2] = q[m * STEP[d]];
        } else {
            w[0] = w[4] = 0.0;
            for (int m = -1; m <= 1; ++m) w[m + 2] = q[m * STEP[d]];
        }
        face_values(c, recon, w, &wm[v], &wp[v]);
    }
}

static int state_ok(const double *W) { return W[0] > 0.0 && W[4] > 0.0; }

/* O4-MHM (Toro 2009 sect. 14.4 / 16.5, MUSCL-Hancock; R6) for cell n */
static void mhm_predict_cell(const ctx_t *c, int recon, double lam_r, const work_t *wk, int n,
                             orc_stats *st)
{
    int nv = c->nv;
    double Wf[3][2][NVMAX], Uf[3][2][NVMAX], Ff[3][2][NVMAX], dU[NVMAX];
    for (int d = 0; d < 3; ++d) {
        gather_face_values(c, recon, wk->W, n, d, Wf[d][0], Wf[d][1]);
        for (int s = 0; s < 2; ++s) {
            prim2cons(c, Wf[d][s], Uf[d][s]);
            phys_flux(c, d, Wf[d][s], Uf[d][s], Ff[d][s]);
        }
    }
    for (int v = 0; v < nv; ++v)
        dU[v] = ((Ff[0][1][v] - Ff[0][0][v]) + (Ff[1][1][v] - Ff[1][0][v])) + (Ff[2][1][v] - Ff[2][0][v]);
    double Ue[3][2][NVMAX];
    int ok = 1;
    for (int d = 0; d < 3; ++d)
        for (int s = 0; s < 2; ++s) {
            double We[NVMAX];
            for (int v = 0; v < nv; ++v) Ue[d][s][v] = Uf[d][s][v] - 0.5 * lam_r * dU[v];
            cons2prim(c, Ue[d][s], We);
            if (floors_set(c)) {
                floor_prim(c, We);
                prim2cons(c, We, Ue[d][s]);
            }
            if (!state_ok(We)) ok = 0;
        }
    if (!ok) st->n_pred_revert++;
    for (int d = 0; d < 3; ++d)
        for (int s = 0; s < 2; ++s)
            for (int v = 0; v < nv; ++v) wk->FS[FSI(d, s, v, n)] = ok ? Ue[d][s][v] : Uf[d][s][v];
}

/* O4-CTU (a) for cell n: traced states, all three axes */
static void ctu_trace_cell(const ctx_t *c, int recon, double lam_r, const work_t *wk, int n,
                           orc_stats *st)
{
    int nv = c->nv;
    double Wc[NVMAX];
    for (int v = 0; v < nv; ++v) Wc[v] = wk->W[(size_t)v * NPC + n];
    for (int d = 0; d < 3; ++d) {
        int in_ = 1 + d, it1 = 1 + (d + 1) % 3, it2 = 1 + (d + 2) % 3;
        double wm[NVMAX], wp[NVMAX];
        gather_face_values(c, recon, wk->W, n, d, wm, wp);
        /* rotate so that the traced axis is "n" */
        double Wr[NVMAX], rm[NVMAX], rp[NVMAX], tm[NVMAX], tp[NVMAX];
        int map[NVMAX] = {0, in_, it1, it2, 4};
        for (int v = 5; v < nv; ++v) map[v] = v;
        for (int v = 0; v < nv; ++v) {
            Wr[v] = Wc[map[v]];
            rm[v] = wm[map[v]];
            rp[v] = wp[map[v]];
        }
        trace_cell(c, recon, Wr, rm, rp, lam_r, tm, tp);
        double Tm[NVMAX], Tp[NVMAX];
        for (int v = 0; v < nv; ++v) {
            Tm[map[v]] = tm[v];
            Tp[map[v]] = tp[v];
        }
        if (floors_set(c)) {
            floor_prim(c, Tm);
            floor_prim(c, Tp);
        }
        if (!state_ok(Tm) || !state_ok(Tp)) { /* R8: revert this axis to the untraced face values */
            st->n_pred_revert++;
            for (int v = 0; v < nv; ++v) {
                Tm[v] = wm[v];
                Tp[v] = wp[v];
            }
        }
        double Um[NVMAX], Up[NVMAX];
        prim2cons(c, Tm, Um);
        prim2cons(c, Tp, Up);
        for (int v = 0; v < nv; ++v) {
            wk->TS[FSI(d, 0, v, n)] = Um[v];
            wk->TS[FSI(d, 1, v, n)] = Up[v];
        }
    }
}

static void face_flux(const ctx_t *c, int solver, int d, const double *S, int n, double *Fout,
                      orc_stats *st)
{
    int nv = c->nv;
    double UL[NVMAX] = {0}, UR[NVMAX] = {0}, F[NVMAX];
    for (int v = 0; v < nv; ++v) {
        UL[v] = S[FSI(d, 1, v, n)];
        UR[v] = S[FSI(d, 0, v, n + STEP[d])];
    }
    riemann(c, solver, d, UL, UR, F, st);
    for (int v = 0; v < nv; ++v) Fout[FLI(d, v, n)] = F[v];
}

/* remedy (ii), L105: first order in space and time, unsplit, same solver (R15) */
static void first_order_cell(const ctx_t *c, int solver, double lam_r, const double *in, int n,
                             double *Unew, orc_stats *st)
{
    int nv = c->nv;
    double Uc[NVMAX], Un[NVMAX], Fm[3][NVMAX], Fp[3][NVMAX];
    for (int v = 0; v < nv; ++v) Uc[v] = in[(size_t)v * NPC + n];
    for (int d = 0; d < 3; ++d) {
        for (int v = 0; v < nv; ++v) Un[v] = in[(size_t)v * NPC + n - STEP[d]];
        riemann(c, solver, d, Un, Uc, Fm[d], st);
        for (int v = 0; v < nv; ++v) Un[v] = in[(size_t)v * NPC + n + STEP[d]];
        riemann(c, solver, d, Uc, Un, Fp[d], st);
    }
    for (int v = 0; v < nv; ++v)
        Unew[v] = Uc[v] - lam_r * (((Fp[0][v] - Fm[0][v]) + (Fp[1][v] - Fm[1][v])) + (Fp[2][v] - Fm[2][v]));
}

static void advance_group(const ctx_t *c, int scheme, int recon, int solver, double dt, double dh,
                          const double *in, double *out, double *flux_out, double *speed_out,
                          work_t *wk, orc_stats *st)
{
    const int nv = c->nv;
    const double lam_r = dt / dh;
    const int lo = NG - 1, hi = NG + PS; /* padded index range of cells -1..16 : [2,19] */

    /* O1 */
    for (int n = 0; n < NPC; ++n) {
        double U[NVMAX], W[NVMAX];
        for (int v = 0; v < nv; ++v) U[v] = in[(size_t)v * NPC + n];
        cons2prim(c, U, W);
        floor_prim(c, W);
        for (int v = 0; v < nv; ++v) wk->W[(size_t)v * NPC + n] = W[v];
    }

    if (scheme == SCHEME_MHM) {
        /* O2-O4: evolved face states of every cell in [-1,16]^3 */
        for (int k = lo; k <= hi; ++k)
            for (int j = lo; j <= hi; ++j)
                for (int i = lo; i <= hi; ++i) mhm_predict_cell(c, recon, lam_r, wk, IDX(i, j, k), st);
    } else if (scheme == SCHEME_VL) {
        /* O4-VL (van Leer 2006; Falle 1991; Stone & Gardiner 2009 sect. 3; reading R26):
         * (a) first-order fluxes: the Riemann solver on the piecewise-constant cell averages, at every face of
         *     the cells [-2,17]^3 (padded [1,20]).  The predictor works on the same floored primitives W as the
         *     reconstruction of the other schemes does (R14): its input states are prim2cons(W). */
        const int l1 = lo - 1, h1 = hi + 1;
        for (int d = 0; d < 3; ++d)
            for (int k = l1 - (d == 2); k <= h1; ++k)
                for (int j = l1 - (d == 1); j <= h1; ++j)
                    for (int i = l1 - (d == 0); i <= h1; ++i) {
                        int n = IDX(i, j, k);
                        double WL[NVMAX], WR[NVMAX], UL[NVMAX] = {0}, UR[NVMAX] = {0}, F[NVMAX];
                        for (int v = 0; v < nv; ++v) {
                            WL[v] = wk->W[(size_t)v * NPC + n];
                            WR[v] = wk->W[(size_t)v * NPC + n + STEP[d]];
                        }
                        prim2cons(c, WL, UL);
                        prim2cons(c, WR, UR);
                        riemann(c, solver, d, UL, UR, F, st);
                        for (int v = 0; v < nv; ++v) wk->F1[FLI(d, v, n)] = F[v];
                    }
        /* (b) half-step state U^{n+1/2} = U^n - dt/(2 dh) sum_d [F1_d(+) - F1_d(-)] of the cells [-2,17]^3, as
         *     primitives; floors if set; an unphysical half-step state falls back to the cell's own U^n */
        for (int k = l1; k <= h1; ++k)
            for (int j = l1; j <= h1; ++j)
                for (int i = l1; i <= h1; ++i) {
                    int n = IDX(i, j, k);
                    double U0[NVMAX], W0[NVMAX], U[NVMAX], W[NVMAX];
                    for (int v = 0; v < nv; ++v) W0[v] = wk->W[(size_t)v * NPC + n];
                    prim2cons(c, W0, U0);
                    for (int v = 0; v < nv; ++v) {
                        double dfx = wk->F1[FLI(0, v, n)] - wk->F1[FLI(0, v, n - STEP[0])];
                        double dfy = wk->F1[FLI(1, v, n)] - wk->F1[FLI(1, v, n - STEP[1])];
                        double dfz = wk->F1[FLI(2, v, n)] - wk->F1[FLI(2, v, n - STEP[2])];
                        U[v] = U0[v] - 0.5 * lam_r * ((dfx + dfy) + dfz);
                    }
                    cons2prim(c, U, W);
                    floor_prim(c, W);
                    if (!state_ok(W)) {
                        st->n_pred_revert++;
                        for (int v = 0; v < nv; ++v) W[v] = W0[v];
                    }
                    for (int v = 0; v < nv; ++v) wk->WH[(size_t)v * NPC + n] = W[v];
                }
        /* (c) face values of the half-step primitives (O2, O3) for every cell of [-1,16]^3, as conserved states */
        for (int k = lo; k <= hi; ++k)
            for (int j = lo; j <= hi; ++j)
                for (int i = lo; i <= hi; ++i) {
                    int n = IDX(i, j, k);
                    for (int d = 0; d < 3; ++d) {
                        double wm[NVMAX], wp[NVMAX], Um[NVMAX], Up[NVMAX];
                        gather_face_values(c, recon, wk->WH, n, d, wm, wp);
                        prim2cons(c, wm, Um);
                        prim2cons(c, wp, Up);
                        for (int v = 0; v < nv; ++v) {
                            wk->FS[FSI(d, 0, v, n)] = Um[v];
                            wk->FS[FSI(d, 1, v, n)] = Up[v];
                        }
                    }
                }
    } else {
        /* (a) traced states */
        for (int k = lo; k <= hi; ++k)
            for (int j = lo; j <= hi; ++j)
                for (int i = lo; i <= hi; ++i) ctu_trace_cell(c, recon, lam_r, wk, IDX(i, j, k), st);
        /* (b) first Riemann pass on every face between two cells of [-1,16]^3 */
        for (int d = 0; d < 3; ++d)
            for (int k = lo; k <= hi - (d == 2); ++k)
                for (int j = lo; j <= hi - (d == 1); ++j)
                    for (int i = lo; i <= hi - (d == 0); ++i)
                        face_flux(c, solver, d, wk->TS, IDX(i, j, k), wk->F1, st);
        /* (c) transverse flux-gradient correction, conserved variables, coefficient 1/2 (R7) */
        for (int d = 0; d < 3; ++d) {
            int d1 = (d + 1) % 3, d2 = (d + 2) % 3;
            int l[3] = {lo + 1, lo + 1, lo + 1}, h[3] = {hi - 1, hi - 1, hi - 1};
            l[d] = lo;
            h[d] = hi;
            for (int k = l[2]; k <= h[2]; ++k)
                for (int j = l[1]; j <= h[1]; ++j)
                    for (int i = l[0]; i <= h[0]; ++i) {
                        int n = IDX(i, j, k);
                        for (int s = 0; s < 2; ++s) {
                            double U[NVMAX], W[NVMAX];
                            for (int v = 0; v < nv; ++v) {
                                double g1 = wk->F1[FLI(d1, v, n)] - wk->F1[FLI(d1, v, n - STEP[d1])];
                                double g2 = wk->F1[FLI(d2, v, n)] - wk->F1[FLI(d2, v, n - STEP[d2])];
                                U[v] = wk->TS[FSI(d, s, v, n)] - 0.5 * lam_r * g1 - 0.5 * lam_r * g2;
                            }
                            cons2prim(c, U, W);
                            if (floors_set(c)) {
                                floor_prim(c, W);
                                prim2cons(c, W, U);
                            }
                            if (!state_ok(W)) { /* R8: keep the uncorrected traced state */
                                st->n_pred_revert++;
                                for (int v = 0; v < nv; ++v) U[v] = wk->TS[FSI(d, s, v, n)];
                            }
                            for (int v = 0; v < nv; ++v) wk->FS[FSI(d, s, v, n)] = U[v];
                        }
                    }
        }
    }

    /* O5: final Riemann pass, faces bounding interior cells */
    for (int d = 0; d < 3; ++d) {
        int l[3] = {NG, NG, NG}, h[3] = {NG + PS - 1, NG + PS - 1, NG + PS - 1};
        l[d] = NG - 1;
        for (int k = l[2]; k <= h[2]; ++k)
            for (int j = l[1]; j <= h[1]; ++j)
                for (int i = l[0]; i <= h[0]; ++i) {
                    int64_t before = st->n_riemann;
                    face_flux(c, solver, d, wk->FS, IDX(i, j, k), wk->FX, st);
                    st->n_riemann_final += st->n_riemann - before;
                }
    }

    /* O6 + O7 */
    double smax = 0.0;
    for (int k = 0; k < PS; ++k)
        for (int j = 0; j < PS; ++j)
            for (int i = 0; i < PS; ++i) {
                int n = IDX(i + NG, j + NG, k + NG);
                double U[NVMAX];
                for (int v = 0; v < nv; ++v) {
                    double dfx = wk->FX[FLI(0, v, n)] - wk->FX[FLI(0, v, n - STEP[0])];
                    double dfy = wk->FX[FLI(1, v, n)] - wk->FX[FLI(1, v, n - STEP[1])];
                    double dfz = wk->FX[FLI(2, v, n)] - wk->FX[FLI(2, v, n - STEP[2])];
                    U[v] = in[(size_t)v * NPC + n] - lam_r * ((dfx + dfy) + dfz);
                }
                dual_energy_fix(c, U, st);
                if (c->o.remedy_first_order && !is_physical(c, U)) {
                    st->n_first_order++;
                    first_order_cell(c, solver, lam_r, in, n, U, st);
                    dual_energy_fix(c, U, st);
                }
                if (floors_set(c)) floor_cons(c, U, st);
                renormalize_scalars(c, U);
                if (!is_physical(c, U)) st->n_unphysical++;
                for (int v = 0; v < nv; ++v) out[(((size_t)v * PS + k) * PS + j) * PS + i] = U[v];
                double s = signal_speed(c, scheme, U);
                if (s > smax) smax = s; /* NaN never wins: comparison false */
            }
    if (speed_out) *speed_out = smax;

    /* O8: boundary fluxes on the patch faces 0, 8, 16 of each axis (L112) */
    if (flux_out) {
        for (int d = 0; d < 3; ++d)
            for (int p = 0; p < 3; ++p)
                for (int v = 0; v < nv; ++v)
                    for (int b = 0; b < PS; ++b)
                        for (int a = 0; a < PS; ++a) {
                            /* (a,b): the two remaining axes, a the faster one */
                            int f = NG - 1 + 8 * p; /* padded index of the cell left of the face */
                            int i, j, k;
                            if (d == 0) { i = f; j = a + NG; k = b + NG; }
                            else if (d == 1) { i = a + NG; j = f; k = b + NG; }
                            else { i = a + NG; j = b + NG; k = f; }
                            flux_out[((((size_t)d * 3 + p) * nv + v) * PS + b) * PS + a] =
                                wk->FX[FLI(d, v, IDX(i, j, k))];
                        }
    }
}

/* ------------------------------------------------------------------------------------------
 * exported entry points
 * ---------------------------------------------------------------------------------------- */
static void make_ctx(ctx_t *c, double gamma, int recon, const orc_opts *o)
{
    c->gamma = gamma;
    c->gm1 = gamma - 1.0;
    if (o) {
        c->o = *o;
    } else {
        memset(&c->o, 0, sizeof(c->o));
        c->o.limiter = LIMITER_GMINMOD;
        c->o.theta = 0.0;
        c->o.de_xi = 1e-2;
    }
    if (c->o.limiter == 0) c->o.limiter = LIMITER_GMINMOD;
    if (!(c->o.theta > 0.0)) c->o.theta = recon == RECON_PPM ? 2.0 : 1.0; /* R3 */
    c->nv = 5 + c->o.n_scalar;
}

int oracle_fluid_advance(const double *in, double *out, double *flux_out, double *group_speed_out,
                         int64_t n_groups, double dt, double dh, double gamma, int scheme, int recon,
                         int riemann_solver, const orc_opts *opts, orc_stats *stats_out)
{
    if (!in || !out || n_groups < 0 || !(dt > 0.0) || !(dh > 0.0) || !(gamma > 1.0)) return -1;
    if (scheme != SCHEME_MHM && scheme != SCHEME_CTU && scheme != SCHEME_VL) return -1;
    if (scheme == SCHEME_VL && recon != RECON_PLM) return -2;   /* VL + PPM needs a fourth ghost zone (L300 fixes three) */
    if (recon != RECON_PLM && recon != RECON_PPM) return -1;
    if (riemann_solver < RSOLVER_ROE || riemann_solver > RSOLVER_EXACT) return -1;
    ctx_t c;
    make_ctx(&c, gamma, recon, opts);
    if (c.o.n_scalar < 0 || c.o.n_scalar > NSMAX) return -1;
    if (c.o.dual_energy && c.o.n_scalar < 1) return -1;
    const int nv = c.nv;
    orc_stats tot;
    memset(&tot, 0, sizeof(tot));
    int fail = 0;
#pragma omp parallel
    {
        work_t wk;
        wk.W = (double *)malloc(sizeof(double) * nv * NPC);
        wk.FS = (double *)malloc(sizeof(double) * 6 * nv * NPC);
        wk.TS = (double *)malloc(sizeof(double) * 6 * nv * NPC);
        wk.F1 = (double *)malloc(sizeof(double) * 3 * nv * NPC);
        wk.FX = (double *)malloc(sizeof(double) * 3 * nv * NPC);
        wk.WH = (double *)malloc(sizeof(double) * nv * NPC);
        orc_stats st;
        memset(&st, 0, sizeof(st));
        if (!wk.W || !wk.FS || !wk.TS || !wk.F1 || !wk.FX || !wk.WH) {
#pragma omp atomic write
            fail = 1;
        } else {
#pragma omp for schedule(dynamic, 1)
            for (int64_t g = 0; g < n_groups; ++g) {
                advance_group(&c, scheme, recon, riemann_solver, dt, dh, in + (size_t)g * nv * NPC,
                              out + (size_t)g * nv * PS * PS * PS,
                              flux_out ? flux_out + (size_t)g * 9 * nv * PS * PS : NULL,
                              group_speed_out ? group_speed_out + g : NULL, &wk, &st);
            }
        }
#pragma omp critical
        {
            tot.n_riemann += st.n_riemann;
            tot.n_riemann_final += st.n_riemann_final;
            tot.n_roe_fallback += st.n_roe_fallback;
            tot.n_pred_revert += st.n_pred_revert;
            tot.n_first_order += st.n_first_order;
            tot.n_dual_fix += st.n_dual_fix;
            tot.n_floor += st.n_floor;
            tot.n_unphysical += st.n_unphysical;
        }
        free(wk.W); free(wk.FS); free(wk.TS); free(wk.F1); free(wk.FX); free(wk.WH);
    }
    if (fail) return -4;
    if (stats_out) *stats_out = tot;
    return 0;
}

/* O9: u is the unpadded state [n_groups][NV][16][16][16];  *dt_out = cfl*dh / max speed */
int oracle_cfl_dt(const double *u, int64_t n_groups, double dh, double gamma, double cfl, int scheme,
                  const orc_opts *opts, double *group_speed_out, double *dt_out)
{
    if (!u || n_groups < 0 || !(dh > 0.0) || !(gamma > 1.0) || !(cfl > 0.0)) return -1;
    ctx_t c;
    make_ctx(&c, gamma, RECON_PLM, opts);
    const int nv = c.nv, nc = PS * PS * PS;
    double gmax = 0.0;
    for (int64_t g = 0; g < n_groups; ++g) {
        double smax = 0.0;
        for (int n = 0; n < nc; ++n) {
            double U[NVMAX];
            for (int v = 0; v < nv; ++v) U[v] = u[((size_t)g * nv + v) * nc + n];
            double s = signal_speed(&c, scheme, U);
            if (s > smax) smax = s;
        }
        if (group_speed_out) group_speed_out[g] = smax;
        if (smax > gmax) gmax = smax;
    }
    if (dt_out) *dt_out = cfl * dh / gmax;
    return 0;
}

/* ---- building blocks exported for the pin tests (each is exactly what the solver calls) ---- */
int oracle_riemann(int solver, int axis, const double *UL, const double *UR, double gamma, int n_scalar,
                   double *F, int *fallback_out)
{
    orc_opts o;
    memset(&o, 0, sizeof(o));
    o.n_scalar = n_scalar;
    ctx_t c;
    make_ctx(&c, gamma, RECON_PLM, &o);
    orc_stats st;
    memset(&st, 0, sizeof(st));
    riemann(&c, solver, axis, UL, UR, F, &st);
    if (fallback_out) *fallback_out = (int)st.n_roe_fallback;
    return 0;
}

/* Roe wave strengths, eigenvalues and right eigenvectors for x-normal states (for the identities
 * sum a_k K_k = dU and sum lambda_k a_k K_k = F_R - F_L on a single jump) */
int oracle_roe_decomposition(const double *UL, const double *UR, double gamma, double *alpha,
                             double *lambda, double *K /* [5][5] */)
{
    ctx_t c;
    make_ctx(&c, gamma, RECON_PLM, NULL);
    rstate_t L, R;
    roeavg_t r;
    rstate(&c, UL, &L);
    rstate(&c, UR, &R);
    roe_average(&c, &L, &R, &r);
    double dU[5];
    for (int v = 0; v < 5; ++v) dU[v] = UR[v] - UL[v];
    double u = r.u, vv = r.v, w = r.w, H = r.H, a = r.a;
    double a3 = dU[2] - vv * dU[0];
    double a4 = dU[3] - w * dU[0];
    double d5 = dU[4] - a3 * vv - a4 * w;
    double a2 = c.gm1 / r.a2 * (dU[0] * (H - u * u) + u * dU[1] - d5);
    double a1 = (dU[0] * (u + a) - dU[1] - a * a2) / (2.0 * a);
    double a5 = dU[0] - (a1 + a2);
    double KK[5][5] = {{1.0, u - a, vv, w, H - u * a},
                       {1.0, u, vv, w, 0.5 * r.q2},
                       {0.0, 0.0, 1.0, 0.0, vv},
                       {0.0, 0.0, 0.0, 1.0, w},
                       {1.0, u + a, vv, w, H + u * a}};
    double al[5] = {a1, a2, a3, a4, a5}, la[5] = {u - a, u, u, u, u + a};
    for (int k = 0; k < 5; ++k) {
        alpha[k] = al[k];
        lambda[k] = la[k];
        for (int v = 0; v < 5; ++v) K[k * 5 + v] = KK[k][v];
    }
    return 0;
}

double oracle_limited_slope(int limiter, double theta, double dL, double dR)
{
    ctx_t c;
    memset(&c, 0, sizeof(c));
    c.o.limiter = limiter;
    c.o.theta = theta;
    return limited_slope(&c, dL, dR);
}

/* face values of cell 2 of a 5-cell strip of one variable */
void oracle_face_values(int recon, int limiter, double theta, const double *w5, double *wm, double *wp)
{
    ctx_t c;
    memset(&c, 0, sizeof(c));
    c.o.limiter = limiter;
    c.o.theta = theta;
    face_values(&c, recon, w5, wm, wp);
}

/* characteristic tracing of one cell: W, wm, wp, tm, tp are x-normal primitive vectors [5+n_scalar] */
void oracle_trace_cell(int recon, double gamma, int n_scalar, const double *W, const double *wm,
                       const double *wp, double dt_over_dh, double *tm, double *tp)
{
    orc_opts o;
    memset(&o, 0, sizeof(o));
    o.n_scalar = n_scalar;
    ctx_t c;
    make_ctx(&c, gamma, recon, &o);
    trace_cell(&c, recon, W, wm, wp, dt_over_dh, tm, tp);
}

/* closing step (dual energy, floors, physical check) of one cell, in place; returns is_physical */
int oracle_close_cell(double *U, double gamma, const orc_opts *opts, orc_stats *st_out)
{
    ctx_t c;
    make_ctx(&c, gamma, RECON_PLM, opts);
    orc_stats st;
    memset(&st, 0, sizeof(st));
    dual_energy_fix(&c, U, &st);
    if (floors_set(&c)) floor_cons(&c, U, &st);
    renormalize_scalars(&c, U);
    if (st_out) *st_out = st;
    return is_physical(&c, U);
}

/* test hook: characteristic-limited slope vector of one cell from the rotated primitive states of cells j-1, j, j+1 */
void oracle_char_slope(int limiter, double theta, double gamma, int n_scalar, const double *Wl, const double *Wc,
                       const double *Wr, double *slope)
{
    orc_opts o;
    memset(&o, 0, sizeof(o));
    o.limiter = limiter;
    o.theta = theta;
    o.n_scalar = n_scalar;
    ctx_t c;
    make_ctx(&c, gamma, RECON_PLM, &o);
    c.o.limiter = limiter;
    c.o.theta = theta;
    char_slope(&c, Wl, Wc, Wr, slope);
}

int oracle_sizeof_opts(void) { return (int)sizeof(orc_opts); }
int oracle_sizeof_stats(void) { return (int)sizeof(orc_stats); }

/* ------------------------------------------------------------------------------------------------
 * The two fix-up operations of PAPER.md L112 between a refined patch group and the coarse level, in the
 * patch-group layout of the solver.  Plain loops, fp64.
 *
 * Restriction: "the data of fine patches are averaged to replace the data of their parent coarse cells".
 * fine[n_fine][nv][16][16][16], coarse[..][nv][16][16][16]; parent[g] = coarse group * 8 + octant,
 * octant = oz*4 + oy*2 + ox: fine group g covers the 8^3 coarse cells of that octant.  The eight children of a
 * coarse cell are summed in the order (dz, dy, dx) = (0,0,0), (0,0,1), (0,1,0), ... and multiplied by 1/8.
 * ---------------------------------------------------------------------------------------------- */
int oracle_restrict(const double *fine, double *coarse, const int32_t *parent, int64_t n_fine, int nv)
{
    for (int64_t g = 0; g < n_fine; ++g) {
        const int64_t cg = parent[g] >> 3;
        const int oz = (parent[g] >> 2) & 1, oy = (parent[g] >> 1) & 1, ox = parent[g] & 1;
        for (int v = 0; v < nv; ++v) {
            const double *f = fine + ((size_t)g * nv + v) * 4096;
            double *c = coarse + ((size_t)cg * nv + v) * 4096;
            for (int k = 0; k < 8; ++k)
                for (int j = 0; j < 8; ++j)
                    for (int i = 0; i < 8; ++i) {
                        double s = 0.0;
                        for (int dz = 0; dz < 2; ++dz)
                            for (int dy = 0; dy < 2; ++dy)
                                for (int dx = 0; dx < 2; ++dx)
                                    s = s + f[((2 * k + dz) * 16 + (2 * j + dy)) * 16 + (2 * i + dx)];
                        c[((oz * 8 + k) * 16 + (oy * 8 + j)) * 16 + (ox * 8 + i)] = 0.125 * s;
                    }
        }
    }
    return 0;
}

/* Flux correction: "the coarse-grid fluxes across the coarse-fine boundaries are replaced by the fine-grid fluxes
 * averaged in space and time" -- applied as a correction of the coarse cells next to the boundary.
 * One table entry = one outer face of a fine group that is a coarse-fine boundary (16 x 16 fine faces = 8 x 8 coarse):
 *   e[0] fine group   e[1] axis d   e[2] side (0: the group's low face, flux plane 0; 1: high face, plane 2)
 *   e[3] coarse group whose flux_out holds the coarse flux there, e[4] its plane (0,1,2),
 *   e[5] (b0 << 8) | a0 : origin of the 8 x 8 quadrant in that 16 x 16 plane (b = slower, a = faster remaining axis)
 *   e[6] coarse group that owns the coarse cells on the other side of the face,
 *   e[7] (z << 16) | (y << 8) | x : the cell of the 8 x 8 patch with b = a = 0 (its coordinate along d is the layer).
 * fine_flux_avg = time average over the coarse step of the fine flux_out; lam = dt_coarse / dh_coarse.
 * U_cell += sgn * lam * (avg2x2(F_fine) - F_coarse), sgn = -1 on side 0 (the face is the cell's upper face), +1 on
 * side 1; avg2x2 = 0.25 * (((f00 + f01) + f10) + f11).  Entries are applied in the order axis 0 side 0, axis 0
 * side 1, axis 1 side 0, ... (within such a pass no two entries touch the same cell). */
int oracle_flux_correct(double *coarse, const double *coarse_flux, const double *fine_flux_avg, const int32_t *tab,
                        int64_t n_entries, int nv, double lam)
{
    for (int pass = 0; pass < 6; ++pass)
        for (int64_t n = 0; n < n_entries; ++n) {
            const int32_t *e = tab + 8 * n;
            const int d = e[1], side = e[2];
            if (d * 2 + side != pass) continue;
            const double sgn = side ? 1.0 : -1.0;
            const int b0 = e[5] >> 8, a0 = e[5] & 255;
            const int z0 = e[7] >> 16, y0 = (e[7] >> 8) & 255, x0 = e[7] & 255;
            for (int v = 0; v < nv; ++v) {
                const double *ff = fine_flux_avg + ((((size_t)e[0] * 3 + d) * 3 + (side ? 2 : 0)) * nv + v) * 256;
                const double *fc = coarse_flux + ((((size_t)e[3] * 3 + d) * 3 + e[4]) * nv + v) * 256;
                double *c = coarse + ((size_t)e[6] * nv + v) * 4096;
                for (int b = 0; b < 8; ++b)
                    for (int a = 0; a < 8; ++a) {
                        const double favg = 0.25 * (((ff[(2 * b) * 16 + 2 * a] + ff[(2 * b) * 16 + 2 * a + 1]) +
                                                     ff[(2 * b + 1) * 16 + 2 * a]) + ff[(2 * b + 1) * 16 + 2 * a + 1]);
                        const double corr = lam * (favg - fc[(b0 + b) * 16 + (a0 + a)]);
                        int z = z0, y = y0, x = x0;
                        if (d == 0) { z += b; y += a; } else if (d == 1) { z += b; x += a; } else { y += b; x += a; }
                        c[(z * 16 + y) * 16 + x] += sgn * corr;
                    }
            }
        }
    return 0;
}
