/*
 * oracle/ppm_oracle.c — TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, fp64 CPU implementation of the one hot path of arxiv/paper_1810_13416
 * (Woodward, Lin, Mao, Andrassy, Herwig): the directionally split 3-D PPM gas-dynamics
 * timestep fused with PPB ten-moment advection of the fractional volume FV
 * (BASELINE.json north_star).
 *
 * The paper prints no equations ("Here we will not repeat the details of these
 * algorithms"), so this file follows, step by step and in the same
 * notation, the readings H0..H9, P1..P4, C1..C7 listed in SURVEY.md section 8(c) and
 * restated in DESIGN.md.  No blocking, fusion or reordering: every step is a loop over
 * a 1-D pencil held in scratch arrays, so it can be checked against the text by eye.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may load this library.  It shares no code, header, table or constant generator
 * with the CUDA path under paper_1810_13416_b200/csrc/ and neither includes the other.
 *
 * Pins (tests/test_oracle_*.py): every routine below is pinned against closed forms,
 * invariants, brute-force quadrature or a textbook exact Riemann solver; the gravity /
 * base-state source terms (base_at, the H6 half-step sources, the H9 time-centred sources,
 * the odd image of g behind a wall, table_lookup off the nodes) by free fall, split
 * invariance, the energy budget and the doubled periodic box (tests/test_oracle_gravity.py).
 * PARITY UNPINNED (no PPMstar code or output exists to compare with): the *constants*
 * of the readings R3 (smoothness ramp 0.1..0.3), R5 (flattening 0.75/10/3/0.05),
 * R7 (5 Newton iterations), R13 (PPB bound B), the choices R1/R11 and the switch-free
 * tracing R8' (its distance from the Colella-Woodward hard-switched tracing is measured
 * in tests/test_oracle_r8prime.py) — they are constrained only by the invariants.
 *
 * Layout: 15 fields per cell, x fastest: 0 rho', 1 ux, 2 uy, 3 uz, 4 p',
 * 5..14 = m000 m100 m010 m001 m200 m020 m002 m110 m101 m011.
 */
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define NG 4     /* ghost cells per side per sweep: "extends outward only 4 cells" PAPER.md L120 */
#define NF 15
#define TINY 1e-30

enum { OR_BC_PERIODIC = 0, OR_BC_REFLECT = 1, OR_BC_OPEN = 2 /* window side: zero-gradient, don't-care */ };
enum { OR_GRAV_NONE = 0, OR_GRAV_CONST_Z = 1, OR_GRAV_RADIAL = 2 };

typedef struct oracle_ctx {
    int n[3];            /* window extent nx, ny, nz */
    int org[3];          /* global index of window cell (0,0,0); 0 for a full grid */
    double dx, gamma, rho_floor, p_floor;
    int grav_kind, grav_n;
    double s0, ds, center[3];
    double *g, *rho0, *p0; /* table nodes (exact copies of the caller's fp32 nodes) */
    int bc[6];           /* xlo xhi ylo yhi zlo zhi */
    double *q[NF];       /* state: perturbation form, no ghosts */
    double *qn[NF];      /* sweep output */
    int flat3d;          /* NEXT-1: fully 3-D shock detector instead of the per-sweep 1-D one */
    double *F3;          /* F~ of every cell (flat3d only), evaluated on the state at the start of the call */
    int sphere;          /* NEXT-3: confining sphere */
    double sph_r, sph_c[3]; /* its radius and centre (physical units) */
    int twofluid;        /* NEXT-4 ("multifluid"): two-fluid equation of state */
    double gamma1, gamma2; /* adiabatic index of the tracked fluid (volume fraction FV) and of the rest */
} oracle_ctx;

static double clamp01(double x) { return fmin(1.0, fmax(0.0, x)); }
static double median3(double a, double b, double c) { return fmax(fmin(a, b), fmin(fmax(a, b), c)); }

/* ------------------------------------------------------------------------------------------
 * C1: base state (rho0, p0, g) from the gravity table, linear interpolation between nodes.
 * ---------------------------------------------------------------------------------------- */
static void table_lookup(const oracle_ctx *c, double s, double *g, double *rho0, double *p0) {
    double t = (s - c->s0) / c->ds;
    int k = (int)floor(t);
    if (k < 0) k = 0;
    if (k > c->grav_n - 2) k = c->grav_n - 2;
    double w = t - (double)k;
    *g = (1.0 - w) * c->g[k] + w * c->g[k + 1];
    *rho0 = (1.0 - w) * c->rho0[k] + w * c->rho0[k + 1];
    *p0 = (1.0 - w) * c->p0[k] + w * c->p0[k + 1];
}

/* base state at the physical point X; gvec = acceleration vector */
static void base_at(const oracle_ctx *c, const double X[3], double *rho0, double *p0, double gvec[3]) {
    gvec[0] = gvec[1] = gvec[2] = 0.0;
    if (c->grav_kind == OR_GRAV_NONE) { *rho0 = 0.0; *p0 = 0.0; return; }
    double g;
    if (c->grav_kind == OR_GRAV_CONST_Z) {
        table_lookup(c, X[2], &g, rho0, p0);
        gvec[2] = g;
        return;
    }
    double r0 = X[0] - c->center[0], r1 = X[1] - c->center[1], r2 = X[2] - c->center[2];
    double r = sqrt(r0 * r0 + r1 * r1 + r2 * r2);
    table_lookup(c, r, &g, rho0, p0);
    if (r > 0.0) { gvec[0] = g * r0 / r; gvec[1] = g * r1 / r; gvec[2] = g * r2 / r; }
}

/* C3: image of cell index i (window-local, may be outside [0,n)) along direction d.
 * Returns the window-local source index and sets *sgn (-1 for a mirror image) and *gpos,
 * the GLOBAL cell index whose position supplies the base state ("ghost cells behind a
 * reflecting wall use the mirror-image interior position", C1). */
static int image_cell(const oracle_ctx *c, int d, int i, int *sgn, int *gpos) {
    int n = c->n[d];
    *sgn = 1;
    if (i >= 0 && i < n) { *gpos = c->org[d] + i; return i; }
    int bc = (i < 0) ? c->bc[2 * d] : c->bc[2 * d + 1];
    if (bc == OR_BC_PERIODIC) { int s = ((i % n) + n) % n; *gpos = c->org[d] + s; return s; }
    if (bc == OR_BC_REFLECT) { int s = (i < 0) ? (-1 - i) : (2 * n - 1 - i); *sgn = -1; *gpos = c->org[d] + s; return s; }
    /* OPEN: zero-gradient data, base state at the ghost's own (true) position */
    *gpos = c->org[d] + i;
    return (i < 0) ? 0 : n - 1;
}

/* image of a face index f (face f = left face of cell f, position f*dx) -> global face index */
static int image_face(const oracle_ctx *c, int d, int f) {
    int n = c->n[d];
    if (f >= 0 && f <= n) {
        /* the periodic seam is ONE face: n wraps to 0 so both cells see the same base state */
        if (f == n && c->bc[2 * d + 1] == OR_BC_PERIODIC) return c->org[d];
        return c->org[d] + f;
    }
    int bc = (f < 0) ? c->bc[2 * d] : c->bc[2 * d + 1];
    if (bc == OR_BC_PERIODIC) return c->org[d] + (((f % n) + n) % n);
    if (bc == OR_BC_REFLECT) return c->org[d] + ((f < 0) ? -f : 2 * n - f);
    return c->org[d] + f;
}

/* ------------------------------------------------------------------------------------------
 * H1: unlimited 4th-order face value between cells ("one order higher").
 *      q^u_{i+1/2} = 7/12 (q_i + q_{i+1}) - 1/12 (q_{i-1} + q_{i+2})
 * ---------------------------------------------------------------------------------------- */
double oracle_h1_face(double qm1, double q0, double qp1, double qp2) {
    return (7.0 / 12.0) * (q0 + qp1) - (1.0 / 12.0) * (qm1 + qp2);
}

/* H2: Colella-Woodward constrained parabola for cell value qi with unlimited faces fl, fr and
 * neighbours qm (i-1), qp (i+1).  Result (ql, qr). */
void oracle_h2_limit(double qm, double qi, double qp, double fl, double fr, double *ql, double *qr) {
    double L = median3(qm, fl, qi);
    double R = median3(qi, fr, qp);
    if ((R - qi) * (qi - L) <= 0.0) { L = qi; R = qi; }
    else {
        double D = R - L, q6 = 6.0 * (qi - 0.5 * (L + R));
        if (D * q6 > D * D) L = 3.0 * qi - 2.0 * R;
        else if (D * q6 < -D * D) R = 3.0 * qi - 2.0 * L;
    }
    *ql = L; *qr = R;
}

/* H3: smoothness measure on the 5-cell stencil i-2..i+2 and its ramp omega. */
double oracle_h3_S(const double q[5]) {
    double d2m = q[2] - 2.0 * q[1] + q[0];
    double d20 = q[3] - 2.0 * q[2] + q[1];
    double d2p = q[4] - 2.0 * q[3] + q[2];
    return fabs(d2p - d2m) / (fabs(d2m) + 2.0 * fabs(d20) + fabs(d2p) + TINY);
}
double oracle_h3_omega(double S) { return clamp01((S - 0.1) / 0.2); }

/* H4: un-spread flattening coefficient f~_i from full pressures p[i-2..i+2] (p5), normal
 * velocities u[i-1], u[i+1] and sound speed c_i.  All switches are continuous ramps. */
double oracle_h4_ftilde(const double p5[5], double um, double up, double ci) {
    double d1 = p5[3] - p5[1], d2 = p5[4] - p5[0];
    double steep = clamp01(10.0 * (fabs(d1) / fmax(fabs(d2), TINY) - 0.75));
    double jump = clamp01(3.0 * fabs(d1) / fmin(p5[3], p5[1]) - 1.0);
    double conv = clamp01((um - up) / (0.05 * ci));
    return steep * jump * conv;
}

/* H5: averages of the parabola (ql, qr, qi) over the rightmost / leftmost fraction sigma. */
double oracle_h5_Fplus(double ql, double qr, double qi, double sigma) {
    double dq = qr - ql, q6 = 6.0 * (qi - 0.5 * (ql + qr));
    return qr - 0.5 * sigma * (dq - (1.0 - 2.0 * sigma / 3.0) * q6);
}
double oracle_h5_Fminus(double ql, double qr, double qi, double sigma) {
    double dq = qr - ql, q6 = 6.0 * (qi - 0.5 * (ql + qr));
    return ql + 0.5 * sigma * (dq + (1.0 - 2.0 * sigma / 3.0) * q6);
}

/* H6: characteristic tracing for one cell.
 * in : ql[5], qr[5], qi[5] parabolas / centre values of (rho', u, v, w, p'); full rho_i, c_i;
 *      dtdx = dt/dx; src[3] = half-step sources for (rho', u, p').
 * out: WL[5] = state left of face i+1/2, WR[5] = state right of face i-1/2, both (rho',u,v,w,p'). */
void oracle_h6_trace(const double ql[5], const double qr[5], const double qi[5], double rho, double c,
                     double dtdx, const double src[3], double WL[5], double WR[5]) {
    const double u = qi[1];
    const double s_m = (u - c) * dtdx, s_0 = u * dtdx, s_p = (u + c) * dtdx;   /* sigma^k = lambda^k dt/dx */
    const double c2 = c * c;
#define FP(k, s) oracle_h5_Fplus(ql[k], qr[k], qi[k], (s))
#define FM(k, s) oracle_h5_Fminus(ql[k], qr[k], qi[k], (s))
    {   /* left of face i+1/2: reference = average over the fastest wave toward the face (u + c) */
        double sp = fmax(s_p, 0.0);
        double rt = FP(0, sp), ut = FP(1, sp), pt = FP(4, sp);
        /* family k in {-, 0}: its own domain of dependence max(sigma^k, 0); a wave that moves AWAY from
         * the face has the zero-width domain F+(.;0) = q_R (reading R8': no hard switch on
         * the sign of lambda^k, so the traced state is a continuous function of the data) */
        double smk = fmax(s_m, 0.0), s0k = fmax(s_0, 0.0);
        double du = ut - FP(1, smk), dp = pt - FP(4, smk);
        double am = (dp - rho * c * du) / (2.0 * c2);
        double dr0 = rt - FP(0, s0k), dp0 = pt - FP(4, s0k);
        double a0 = dr0 - dp0 / c2;
        WL[0] = rt - am - a0;
        WL[1] = ut + (c / rho) * am;
        WL[4] = pt - c2 * am;
        WL[2] = FP(2, s0k);
        WL[3] = FP(3, s0k);
    }
    {   /* right of face i-1/2: reference = average over the domain of u - c */
        double sm = fmax(-s_m, 0.0);
        double rt = FM(0, sm), ut = FM(1, sm), pt = FM(4, sm);
        double spk = fmax(-s_p, 0.0), s0k = fmax(-s_0, 0.0);
        double du = ut - FM(1, spk), dp = pt - FM(4, spk);
        double ap = (dp + rho * c * du) / (2.0 * c2);
        double dr0 = rt - FM(0, s0k), dp0 = pt - FM(4, s0k);
        double a0 = dr0 - dp0 / c2;
        WR[0] = rt - ap - a0;
        WR[1] = ut - (c / rho) * ap;
        WR[4] = pt - c2 * ap;
        WR[2] = FM(2, s0k);
        WR[3] = FM(3, s0k);
    }
#undef FP
#undef FM
    WL[0] += src[0]; WL[1] += src[1]; WL[4] += src[2];
    WR[0] += src[0]; WR[1] += src[1]; WR[4] += src[2];
}

/* H7: two-shock approximate Riemann solver, FIXED 5 Newton iterations from the acoustic guess,
 * sampled at x/t = 0.  L[5], R[5] = full (rho, u, v, w, p).  out[5] = (rho^, u^, v^, w^, p^);
 * returns p* through *pstar and u* through *ustar when non-NULL. */
void oracle_h7_riemann(const double L[5], const double R[5], double gamma, double rho_floor, double p_floor,
                       double out[5], double *pstar_out, double *ustar_out) {
    const double rl = L[0], ul = L[1], pl = L[4], rr = R[0], ur = R[1], pr = R[4];
    const double CL = sqrt(gamma * pl * rl), CR = sqrt(gamma * pr * rr);
    const double gp = 0.5 * (gamma + 1.0), gm = 0.5 * (gamma - 1.0);
    double ps = fmax(p_floor, (CR * pl + CL * pr + CL * CR * (ul - ur)) / (CL + CR));
    double WL, WR;
    for (int it = 0; it < 5; ++it) {
        WL = sqrt(rl * (gp * ps + gm * pl));
        WR = sqrt(rr * (gp * ps + gm * pr));
        double usl = ul - (ps - pl) / WL;
        double usr = ur + (ps - pr) / WR;
        double ZL = 2.0 * WL * WL * WL / (WL * WL + CL * CL);
        double ZR = 2.0 * WR * WR * WR / (WR * WR + CR * CR);
        ps = fmax(p_floor, ps - ZL * ZR * (usr - usl) / (ZL + ZR));
    }
    WL = sqrt(rl * (gp * ps + gm * pl));
    WR = sqrt(rr * (gp * ps + gm * pr));
    const double us = (WL * ul + WR * ur + pl - pr) / (WL + WR);
    if (pstar_out) *pstar_out = ps;
    if (ustar_out) *ustar_out = us;

    /* sampling at x/t = 0 in the frame mirrored so that the upwind side K is on the left */
    double s, rK, uK, pK, WK;
    const double *K;
    if (us >= 0.0) { s = 1.0; K = L; rK = rl; uK = ul; pK = pl; WK = WL; }
    else           { s = -1.0; K = R; rK = rr; uK = ur; pK = pr; WK = WR; }
    double rs = 1.0 / (1.0 / rK - (ps - pK) / (WK * WK));
    rs = fmax(rs, rho_floor);
    const double cK = sqrt(gamma * pK / rK), cs = sqrt(gamma * ps / rs);
    const double uKh = s * uK, ush = s * us;
    double lam_head, lam_tail;
    if (ps > pK) { lam_head = lam_tail = uKh - WK / rK; }
    else { lam_head = uKh - cK; lam_tail = ush - cs; }
    double th;
    if (lam_head >= 0.0) th = 0.0;
    else if (lam_tail <= 0.0) th = 1.0;
    else th = -lam_head / (lam_tail - lam_head);
    out[0] = (1.0 - th) * rK + th * rs;
    out[1] = (1.0 - th) * uK + th * us;
    out[4] = (1.0 - th) * pK + th * ps;
    out[2] = K[2];
    out[3] = K[3];
}

/* ------------------------------------------------------------------------------------------
 * PPB.  Basis P0 = 1, P1 = s, P2 = s^2 - 1/12 on [-1/2, 1/2]; norms 1, 1/12, 1/180 (C1).
 * ---------------------------------------------------------------------------------------- */
static const double PPB_NORM[3] = {1.0, 1.0 / 12.0, 1.0 / 180.0};
static double ppb_P(int n, double s) { return n == 0 ? 1.0 : (n == 1 ? s : s * s - 1.0 / 12.0); }

/* P2: bound-preserving scaling theta of the nine higher coefficients. */
double oracle_p2_theta(const double m[10]) {
    double B = 0.5 * (fabs(m[1]) + fabs(m[2]) + fabs(m[3]))
             + (1.0 / 6.0) * (fabs(m[4]) + fabs(m[5]) + fabs(m[6]))
             + 0.25 * (fabs(m[7]) + fabs(m[8]) + fabs(m[9]));
    return fmin(1.0, fmax(0.0, fmin(m[0], 1.0 - m[0])) / fmax(B, TINY));
}

/* P4: remap of ONE family (degree deg) for ONE new cell.
 * a[3][3]: coefficients (a0,a1,a2) of the donor cells i-1, i, i+1 (already pre-limited);
 * M[3]: their masses; dMl = mass through the left face i-1/2 (>0: rightward), dMr at i+1/2.
 * out[0..deg] = new coefficients.  Returns 0 if the new mass is <= tiny (cell left unchanged). */
int oracle_p4_remap(int deg, const double a[3][3], const double M[3], double dMl, double dMr, double out[3]) {
    const double Mn = M[1] - dMr + dMl;
    if (Mn <= TINY) { for (int n = 0; n <= deg; ++n) out[n] = a[1][n]; return 0; }
    int src[3]; double slo[3], shi[3]; int np = 0;
    if (dMl > 0.0) { double sg = dMl / M[0]; src[np] = 0; slo[np] = 0.5 - sg; shi[np] = 0.5; ++np; }
    src[np] = 1; slo[np] = -0.5 + fmax(-dMl, 0.0) / M[1]; shi[np] = 0.5 - fmax(dMr, 0.0) / M[1]; ++np;
    if (dMr < 0.0) { double sg = -dMr / M[2]; src[np] = 2; slo[np] = -0.5; shi[np] = -0.5 + sg; ++np; }
    static const double GX[3] = {-0.38729833462074168852, 0.0, 0.38729833462074168852}; /* sqrt(3/5)/2 */
    static const double GW[3] = {5.0 / 18.0, 8.0 / 18.0, 5.0 / 18.0};
    double acc[3] = {0.0, 0.0, 0.0};
    double spos = -0.5;
    for (int k = 0; k < np; ++k) {
        const double *ak = a[src[k]];
        double wk = (shi[k] - slo[k]) * M[src[k]] / Mn;   /* width in the new mass coordinate */
        for (int g = 0; g < 3; ++g) {
            double sn = spos + wk * (0.5 + GX[g]);
            double so = slo[k] + (shi[k] - slo[k]) * (0.5 + GX[g]);
            double qv = ak[0] + ak[1] * so + ak[2] * (so * so - 1.0 / 12.0);
            for (int n = 0; n <= deg; ++n) acc[n] += wk * GW[g] * qv * ppb_P(n, sn);
        }
        spos += wk;
    }
    for (int n = 0; n <= deg; ++n) out[n] = acc[n] / PPB_NORM[n];
    return 1;
}

/* P3: families per sweep direction.  FAM[d][f] = {degree, idx a0, idx a1, idx a2} into m[10]. */
static const int PPB_FAM[3][6][4] = {
    /* x */ {{2, 0, 1, 4}, {1, 2, 7, -1}, {1, 3, 8, -1}, {0, 5, -1, -1}, {0, 6, -1, -1}, {0, 9, -1, -1}},
    /* y */ {{2, 0, 2, 5}, {1, 1, 7, -1}, {1, 3, 9, -1}, {0, 4, -1, -1}, {0, 6, -1, -1}, {0, 8, -1, -1}},
    /* z */ {{2, 0, 3, 6}, {1, 1, 8, -1}, {1, 2, 9, -1}, {0, 4, -1, -1}, {0, 5, -1, -1}, {0, 7, -1, -1}}};
/* coefficients odd in the normal direction (C3) */
static int ppb_is_odd(int d, int k) {
    for (int f = 0; f < 3; ++f) if (PPB_FAM[d][f][2] == k) return 1;
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * C4 + C5: one pencil, direction d.  All input arrays have n + 2*NG entries (cell j = i + NG);
 * face arrays n + 2*NG + 1 (face f = left face of cell j = f).  q[0..4] = rho', u(normal), v, w, p';
 * m[0..9] PPB coefficients in STORAGE order.  Outputs have n entries.
 * ---------------------------------------------------------------------------------------- */
void oracle_sweep_pencil(int n, int d, double dx, double dt, double gamma, double rho_floor, double p_floor,
                         const double *const q[5], const double *const m[10],
                         const double *rho0c, const double *p0c, const double *gd,
                         const double *rho0f, const double *p0f,
                         double *const qn[5], double *const mn[10], const double *ft_ext) {
    const int nt = n + 2 * NG;
    const double dtdx = dt / dx;
    double *buf = (double *)calloc((size_t)nt * 40 + 64, sizeof(double));
    double *rho = buf, *p = rho + nt, *c = p + nt, *ft = c + nt, *fl = ft + nt;
    double *qu[5], *ql[5], *qr[5], *WL[5], *WR[5], *F[5];
    double *cur = fl + nt;
    for (int k = 0; k < 5; ++k) { qu[k] = cur; cur += nt + 1; }
    for (int k = 0; k < 5; ++k) { ql[k] = cur; cur += nt; }
    for (int k = 0; k < 5; ++k) { qr[k] = cur; cur += nt; }
    for (int k = 0; k < 5; ++k) { WL[k] = cur; cur += nt; }
    for (int k = 0; k < 5; ++k) { WR[k] = cur; cur += nt; }
    for (int k = 0; k < 5; ++k) { F[k] = cur; cur += nt + 1; }
    double *dM = cur; cur += nt + 1;
    double *theta = cur; cur += nt;

    /* H0 */
    for (int j = 0; j < nt; ++j) {
        rho[j] = rho0c[j] + q[0][j];
        p[j] = p0c[j] + q[4][j];
        c[j] = sqrt(gamma * p[j] / rho[j]);
    }
    /* H1: face f between cells f-1 and f, for the faces of cells 3 .. nt-4 */
    for (int f = 3; f <= nt - 3; ++f)
        for (int k = 0; k < 5; ++k) qu[k][f] = oracle_h1_face(q[k][f - 2], q[k][f - 1], q[k][f], q[k][f + 1]);
    /* H4: f~ then spread */
    for (int j = 2; j <= nt - 3; ++j) {
        double p5[5] = {p[j - 2], p[j - 1], p[j], p[j + 1], p[j + 2]};
        ft[j] = oracle_h4_ftilde(p5, q[1][j - 1], q[1][j + 1], c[j]);
        /* NEXT-1 ("fully 3-D"): the un-spread coefficient comes from the 3-D detector field instead */
        if (ft_ext) ft[j] = ft_ext[j];
    }
    for (int j = 3; j <= nt - 4; ++j) fl[j] = fmax(ft[j - 1], fmax(ft[j], ft[j + 1]));
    /* H2, H3, H4 applied: parabolas of cells 3 .. nt-4 */
    for (int j = 3; j <= nt - 4; ++j)
        for (int k = 0; k < 5; ++k) {
            double Lm, Rm;
            oracle_h2_limit(q[k][j - 1], q[k][j], q[k][j + 1], qu[k][j], qu[k][j + 1], &Lm, &Rm);
            double q5[5] = {q[k][j - 2], q[k][j - 1], q[k][j], q[k][j + 1], q[k][j + 2]};
            double om = oracle_h3_omega(oracle_h3_S(q5));
            double L = (1.0 - om) * qu[k][j] + om * Lm;
            double R = (1.0 - om) * qu[k][j + 1] + om * Rm;
            ql[k][j] = fl[j] * q[k][j] + (1.0 - fl[j]) * L;
            qr[k][j] = fl[j] * q[k][j] + (1.0 - fl[j]) * R;
        }
    /* H5, H6: traced states of cells 3 .. nt-4 */
    for (int j = 3; j <= nt - 4; ++j) {
        double a[5], b[5], ci[5], wl[5], wr[5], src[3];
        for (int k = 0; k < 5; ++k) { a[k] = ql[k][j]; b[k] = qr[k][j]; ci[k] = q[k][j]; }
        src[0] = 0.5 * dt * (-q[1][j] * (rho0f[j + 1] - rho0f[j]) / dx);
        src[2] = 0.5 * dt * (-q[1][j] * (p0f[j + 1] - p0f[j]) / dx);
        src[1] = 0.5 * dt * gd[j] * q[0][j] / rho[j];
        oracle_h6_trace(a, b, ci, rho[j], c[j], dtdx, src, wl, wr);
        for (int k = 0; k < 5; ++k) { WL[k][j] = wl[k]; WR[k][j] = wr[k]; }
    }
    /* H7, H8: faces f = NG .. nt-NG (between cells f-1 and f) */
    for (int f = NG; f <= nt - NG; ++f) {
        double L[5], R[5], o[5];
        L[0] = fmax(rho0f[f] + WL[0][f - 1], rho_floor); R[0] = fmax(rho0f[f] + WR[0][f], rho_floor);
        L[4] = fmax(p0f[f] + WL[4][f - 1], p_floor);     R[4] = fmax(p0f[f] + WR[4][f], p_floor);
        for (int k = 1; k <= 3; ++k) { L[k] = WL[k][f - 1]; R[k] = WR[k][f]; }
        oracle_h7_riemann(L, R, gamma, rho_floor, p_floor, o, NULL, NULL);
        double Fm = o[0] * o[1];
        double pprime = o[4] - p0f[f];
        F[0][f] = Fm;
        F[1][f] = Fm * o[1] + pprime;
        F[2][f] = Fm * o[2];
        F[3][f] = Fm * o[3];
        F[4][f] = o[1] * (gamma / (gamma - 1.0) * o[4] + 0.5 * o[0] * (o[1] * o[1] + o[2] * o[2] + o[3] * o[3]));
        dM[f] = dt * Fm;     /* P1 */
    }
    /* H9 */
    for (int j = NG; j < nt - NG; ++j) {
        const int i = j - NG;
        const double r0 = rho[j], u0 = q[1][j], v0 = q[2][j], w0 = q[3][j];
        const double E0 = p[j] / (gamma - 1.0) + 0.5 * r0 * (u0 * u0 + v0 * v0 + w0 * w0);
        double r1 = r0 - dtdx * (F[0][j + 1] - F[0][j]);
        r1 = fmax(r1, rho_floor);
        const double rp1 = r1 - rho0c[j];
        const double mu0 = r0 * u0;
        const double mu1 = mu0 - dtdx * (F[1][j + 1] - F[1][j]) + dt * 0.5 * (q[0][j] + rp1) * gd[j];
        const double mv1 = r0 * v0 - dtdx * (F[2][j + 1] - F[2][j]);
        const double mw1 = r0 * w0 - dtdx * (F[3][j + 1] - F[3][j]);
        const double E1 = E0 - dtdx * (F[4][j + 1] - F[4][j]) + dt * 0.5 * (mu0 + mu1) * gd[j];
        const double u1 = mu1 / r1, v1 = mv1 / r1, w1 = mw1 / r1;
        const double p1 = fmax(p_floor, (gamma - 1.0) * (E1 - 0.5 * r1 * (u1 * u1 + v1 * v1 + w1 * w1)));
        qn[0][i] = rp1; qn[1][i] = u1; qn[2][i] = v1; qn[3][i] = w1; qn[4][i] = p1 - p0c[j];
    }
    /* P2 for cells 3 .. nt-4 */
    for (int j = 3; j <= nt - 4; ++j) {
        double mm[10];
        for (int k = 0; k < 10; ++k) mm[k] = m[k][j];
        theta[j] = oracle_p2_theta(mm);
    }
    /* P1, P3, P4 */
    for (int j = NG; j < nt - NG; ++j) {
        const int i = j - NG;
        double M[3] = {rho[j - 1] * dx, rho[j] * dx, rho[j + 1] * dx};
        for (int f = 0; f < 6; ++f) {
            const int deg = PPB_FAM[d][f][0];
            double a[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}}, out[3];
            for (int s = 0; s < 3; ++s)
                for (int nn = 0; nn <= deg; ++nn) {
                    int idx = PPB_FAM[d][f][1 + nn];
                    double v = m[idx][j - 1 + s];
                    if (idx != 0) v *= theta[j - 1 + s];
                    a[s][nn] = v;
                }
            int ok = oracle_p4_remap(deg, a, M, dM[j], dM[j + 1], out);
            for (int nn = 0; nn <= deg; ++nn) {
                int idx = PPB_FAM[d][f][1 + nn];
                mn[idx][i] = ok ? out[nn] : m[idx][j];
            }
        }
    }
    free(buf);
}

/* ------------------------------------------------------------------------------------------
 * NEXT-4 ("multifluid", L87 "fv ... gives the fraction of the volume of a cell that
 * is occupied by a special, tracked multifluid constituent"): two-fluid equation of state.  The paper prints no
 * EOS, so this is reading R25:
 *   the tracked fluid (volume fraction f = FV) and the rest are ideal gases with adiabatic indices gamma1 and
 *   gamma2 in pressure equilibrium inside a cell, so the internal energy per volume is
 *       e = f p/(gamma1-1) + (1-f) p/(gamma2-1) = p beta(f),   beta(f) = f/(gamma1-1) + (1-f)/(gamma2-1),
 *   i.e. the cell behaves as an ideal gas with Gamma(f) = 1 + 1/beta(f), and f is the PPB cell mean m000
 *   clamped to [0,1].  Everything else is the single-fluid scheme with gamma -> Gamma of the cell it belongs to:
 *   c_i = sqrt(Gamma_i p_i/rho_i) (H0, used by H4 and H6); the Riemann problem at a face takes Gamma of its left
 *   cell for the left state and of its right cell for the right state (H7: the contact separates them); the
 *   energy flux carries the enthalpy (beta~ + 1) p^ of the gas that actually crosses the face: beta~ = beta(f~), f~ =
 *   the mean FV of the slab of mass dM that the PPB remap donates through that face (H8) — so the energy flux and
 *   the FV flux move the same gas; and the new pressure is recovered from the conserved energy with beta of the NEW
 *   f, i.e. after this sweep's PPB remap (H9: p = (E - KE)/beta(f_new)).  Total energy sum(p beta(f) + KE) is
 *   conserved to round-off; a contact at rest in pressure equilibrium stays exactly so; a contact carried by a
 *   uniform flow of uniform density keeps its pressure to round-off (with the upwind CELL-MEAN Gamma in the
 *   enthalpy instead, a two-gas shock tube grows an O(1) density spike at the contact and does not converge: tried,
 *   measured, rejected); with gamma1 = gamma2 the scheme is the single-fluid one.
 *   (Remaining limit: FV is remapped in the MASS coordinate (R11), beta is a VOLUME average; across a contact that is
 *   also a density jump the two differ and a moving contact keeps a small pressure ripple, quantified in
 *   tests/test_oracle_twofluid.py.)
 * ---------------------------------------------------------------------------------------- */
double oracle_mix_beta(double f, double gamma1, double gamma2) {
    f = clamp01(f);
    return f / (gamma1 - 1.0) + (1.0 - f) / (gamma2 - 1.0);
}
double oracle_mix_gamma(double f, double gamma1, double gamma2) { return 1.0 + 1.0 / oracle_mix_beta(f, gamma1, gamma2); }

/* H7 with one adiabatic index per side; *gam_out = the index of the side the sampled state lies on */
void oracle_h7_riemann_2f(const double L[5], const double R[5], double gamL, double gamR, double rho_floor, double p_floor,
                          double out[5], double *gam_out, double *pstar_out, double *ustar_out) {
    const double rl = L[0], ul = L[1], pl = L[4], rr = R[0], ur = R[1], pr = R[4];
    const double CL = sqrt(gamL * pl * rl), CR = sqrt(gamR * pr * rr);
    const double gpL = 0.5 * (gamL + 1.0), gmL = 0.5 * (gamL - 1.0), gpR = 0.5 * (gamR + 1.0), gmR = 0.5 * (gamR - 1.0);
    double ps = fmax(p_floor, (CR * pl + CL * pr + CL * CR * (ul - ur)) / (CL + CR));
    double WL, WR;
    for (int it = 0; it < 5; ++it) {
        WL = sqrt(rl * (gpL * ps + gmL * pl));
        WR = sqrt(rr * (gpR * ps + gmR * pr));
        double usl = ul - (ps - pl) / WL;
        double usr = ur + (ps - pr) / WR;
        double ZL = 2.0 * WL * WL * WL / (WL * WL + CL * CL);
        double ZR = 2.0 * WR * WR * WR / (WR * WR + CR * CR);
        ps = fmax(p_floor, ps - ZL * ZR * (usr - usl) / (ZL + ZR));
    }
    WL = sqrt(rl * (gpL * ps + gmL * pl));
    WR = sqrt(rr * (gpR * ps + gmR * pr));
    const double us = (WL * ul + WR * ur + pl - pr) / (WL + WR);
    if (pstar_out) *pstar_out = ps;
    if (ustar_out) *ustar_out = us;
    double s, rK, uK, pK, WK, gK;
    const double *K;
    if (us >= 0.0) { s = 1.0; K = L; rK = rl; uK = ul; pK = pl; WK = WL; gK = gamL; }
    else           { s = -1.0; K = R; rK = rr; uK = ur; pK = pr; WK = WR; gK = gamR; }
    double rs = 1.0 / (1.0 / rK - (ps - pK) / (WK * WK));
    rs = fmax(rs, rho_floor);
    const double cK = sqrt(gK * pK / rK), cs = sqrt(gK * ps / rs);
    const double uKh = s * uK, ush = s * us;
    double lam_head, lam_tail;
    if (ps > pK) { lam_head = lam_tail = uKh - WK / rK; }
    else { lam_head = uKh - cK; lam_tail = ush - cs; }
    double th;
    if (lam_head >= 0.0) th = 0.0;
    else if (lam_tail <= 0.0) th = 1.0;
    else th = -lam_head / (lam_tail - lam_head);
    out[0] = (1.0 - th) * rK + th * rs;
    out[1] = (1.0 - th) * uK + th * us;
    out[4] = (1.0 - th) * pK + th * ps;
    out[2] = K[2];
    out[3] = K[3];
    *gam_out = gK;
}

/* C4 + C5 for the two-fluid EOS: oracle_sweep_pencil step by step, with Gamma of the cell / side in place of gamma
 * and the pressure taken from the energy AFTER the PPB remap (same arguments, same array conventions). */
void oracle_sweep_pencil_2f(int n, int d, double dx, double dt, double gamma1, double gamma2, double rho_floor, double p_floor,
                            const double *const q[5], const double *const m[10],
                            const double *rho0c, const double *p0c, const double *gd,
                            const double *rho0f, const double *p0f,
                            double *const qn[5], double *const mn[10], const double *ft_ext) {
    const int nt = n + 2 * NG;
    const double dtdx = dt / dx;
    double *buf = (double *)calloc((size_t)nt * 43 + 64, sizeof(double));
    double *rho = buf, *p = rho + nt, *c = p + nt, *ft = c + nt, *fl = ft + nt;
    double *qu[5], *ql[5], *qr[5], *WL[5], *WR[5], *F[5];
    double *cur = fl + nt;
    for (int k = 0; k < 5; ++k) { qu[k] = cur; cur += nt + 1; }
    for (int k = 0; k < 5; ++k) { ql[k] = cur; cur += nt; }
    for (int k = 0; k < 5; ++k) { qr[k] = cur; cur += nt; }
    for (int k = 0; k < 5; ++k) { WL[k] = cur; cur += nt; }
    for (int k = 0; k < 5; ++k) { WR[k] = cur; cur += nt; }
    for (int k = 0; k < 5; ++k) { F[k] = cur; cur += nt + 1; }
    double *dM = cur; cur += nt + 1;
    double *theta = cur; cur += nt;
    double *Gam = cur; cur += nt;          /* Gamma(f_i) of every cell, from the PPB cell mean the sweep starts from */
    double *E1 = cur; cur += nt;           /* new total energy of the interior cells */
    double *KE1 = cur; cur += nt;          /* their new kinetic energy */

    /* H0 */
    for (int j = 0; j < nt; ++j) {
        Gam[j] = oracle_mix_gamma(m[0][j], gamma1, gamma2);
        rho[j] = rho0c[j] + q[0][j];
        p[j] = p0c[j] + q[4][j];
        c[j] = sqrt(Gam[j] * p[j] / rho[j]);
    }
    /* H1 */
    for (int f = 3; f <= nt - 3; ++f)
        for (int k = 0; k < 5; ++k) qu[k][f] = oracle_h1_face(q[k][f - 2], q[k][f - 1], q[k][f], q[k][f + 1]);
    /* H4 */
    for (int j = 2; j <= nt - 3; ++j) {
        double p5[5] = {p[j - 2], p[j - 1], p[j], p[j + 1], p[j + 2]};
        ft[j] = oracle_h4_ftilde(p5, q[1][j - 1], q[1][j + 1], c[j]);
        if (ft_ext) ft[j] = ft_ext[j];
    }
    for (int j = 3; j <= nt - 4; ++j) fl[j] = fmax(ft[j - 1], fmax(ft[j], ft[j + 1]));
    /* H2, H3, H4 applied */
    for (int j = 3; j <= nt - 4; ++j)
        for (int k = 0; k < 5; ++k) {
            double Lm, Rm;
            oracle_h2_limit(q[k][j - 1], q[k][j], q[k][j + 1], qu[k][j], qu[k][j + 1], &Lm, &Rm);
            double q5[5] = {q[k][j - 2], q[k][j - 1], q[k][j], q[k][j + 1], q[k][j + 2]};
            double om = oracle_h3_omega(oracle_h3_S(q5));
            double L = (1.0 - om) * qu[k][j] + om * Lm;
            double R = (1.0 - om) * qu[k][j + 1] + om * Rm;
            ql[k][j] = fl[j] * q[k][j] + (1.0 - fl[j]) * L;
            qr[k][j] = fl[j] * q[k][j] + (1.0 - fl[j]) * R;
        }
    /* H5, H6 (the cell's own sound speed c_i carries Gamma_i) */
    for (int j = 3; j <= nt - 4; ++j) {
        double a[5], b[5], ci[5], wl[5], wr[5], src[3];
        for (int k = 0; k < 5; ++k) { a[k] = ql[k][j]; b[k] = qr[k][j]; ci[k] = q[k][j]; }
        src[0] = 0.5 * dt * (-q[1][j] * (rho0f[j + 1] - rho0f[j]) / dx);
        src[2] = 0.5 * dt * (-q[1][j] * (p0f[j + 1] - p0f[j]) / dx);
        src[1] = 0.5 * dt * gd[j] * q[0][j] / rho[j];
        oracle_h6_trace(a, b, ci, rho[j], c[j], dtdx, src, wl, wr);
        for (int k = 0; k < 5; ++k) { WL[k][j] = wl[k]; WR[k][j] = wr[k]; }
    }
    /* P2 (ahead of H8, which needs the pre-limited polynomial of the donor cell) */
    for (int j = 3; j <= nt - 4; ++j) {
        double mm[10];
        for (int k = 0; k < 10; ++k) mm[k] = m[k][j];
        theta[j] = oracle_p2_theta(mm);
    }
    /* H7, H8: face f lies between cells f-1 (Gamma_L) and f (Gamma_R) */
    for (int f = NG; f <= nt - NG; ++f) {
        double L[5], R[5], o[5], gh;
        L[0] = fmax(rho0f[f] + WL[0][f - 1], rho_floor); R[0] = fmax(rho0f[f] + WR[0][f], rho_floor);
        L[4] = fmax(p0f[f] + WL[4][f - 1], p_floor);     R[4] = fmax(p0f[f] + WR[4][f], p_floor);
        for (int k = 1; k <= 3; ++k) { L[k] = WL[k][f - 1]; R[k] = WR[k][f]; }
        oracle_h7_riemann_2f(L, R, Gam[f - 1], Gam[f], rho_floor, p_floor, o, &gh, NULL, NULL);
        (void)gh;            /* (Gamma of the sampled side: the sound speeds inside the solver have used it) */
        double Fm = o[0] * o[1];
        double pprime = o[4] - p0f[f];
        F[0][f] = Fm;
        F[1][f] = Fm * o[1] + pprime;
        F[2][f] = Fm * o[2];
        F[3][f] = Fm * o[3];
        dM[f] = dt * Fm;     /* P1 */
        /* the enthalpy that crosses the face belongs to the gas that crosses it: beta of the mean FV of the slab of mass
         * dM that the PPB remap takes out of the donor cell (its pre-limited polynomial along the sweep, P2/P4; the
         * transverse families average to zero over the slab).  With this the internal-energy flux p^ u^ beta~ and the
         * FV flux of the remap move the SAME gas, and a contact carried by a uniform flow of uniform density keeps
         * its pressure exactly. */
        {
            const int jd = (dM[f] >= 0.0) ? f - 1 : f;                       /* donor cell */
            const double sig = fmin(fabs(dM[f]) / (rho[jd] * dx), 1.0);      /* donated fraction of its mass */
            const double sm = (dM[f] >= 0.0) ? 0.5 - 0.5 * sig : -0.5 + 0.5 * sig;   /* slab midpoint in the cell's mass coordinate */
            const int i1 = PPB_FAM[d][0][2], i2 = PPB_FAM[d][0][3];
            const double fs = m[0][jd] + theta[jd] * (m[i1][jd] * sm + m[i2][jd] * (sm * sm + sig * sig / 12.0 - 1.0 / 12.0));
            const double bh = oracle_mix_beta(fs, gamma1, gamma2);
            F[4][f] = o[1] * ((bh + 1.0) * o[4] + 0.5 * o[0] * (o[1] * o[1] + o[2] * o[2] + o[3] * o[3]));
        }
    }
    /* H9, first part: density, momenta and the conserved energy (E0 with beta of the OLD f) */
    for (int j = NG; j < nt - NG; ++j) {
        const int i = j - NG;
        const double r0 = rho[j], u0 = q[1][j], v0 = q[2][j], w0 = q[3][j];
        const double E0 = p[j] / (Gam[j] - 1.0) + 0.5 * r0 * (u0 * u0 + v0 * v0 + w0 * w0);
        double r1 = r0 - dtdx * (F[0][j + 1] - F[0][j]);
        r1 = fmax(r1, rho_floor);
        const double rp1 = r1 - rho0c[j];
        const double mu0 = r0 * u0;
        const double mu1 = mu0 - dtdx * (F[1][j + 1] - F[1][j]) + dt * 0.5 * (q[0][j] + rp1) * gd[j];
        const double mv1 = r0 * v0 - dtdx * (F[2][j + 1] - F[2][j]);
        const double mw1 = r0 * w0 - dtdx * (F[3][j + 1] - F[3][j]);
        E1[j] = E0 - dtdx * (F[4][j + 1] - F[4][j]) + dt * 0.5 * (mu0 + mu1) * gd[j];
        const double u1 = mu1 / r1, v1 = mv1 / r1, w1 = mw1 / r1;
        KE1[j] = 0.5 * r1 * (u1 * u1 + v1 * v1 + w1 * w1);
        qn[0][i] = rp1; qn[1][i] = u1; qn[2][i] = v1; qn[3][i] = w1;
    }
    /* P1, P3, P4 */
    for (int j = NG; j < nt - NG; ++j) {
        const int i = j - NG;
        double M[3] = {rho[j - 1] * dx, rho[j] * dx, rho[j + 1] * dx};
        for (int f = 0; f < 6; ++f) {
            const int deg = PPB_FAM[d][f][0];
            double a[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}}, out[3];
            for (int s = 0; s < 3; ++s)
                for (int nn = 0; nn <= deg; ++nn) {
                    int idx = PPB_FAM[d][f][1 + nn];
                    double v = m[idx][j - 1 + s];
                    if (idx != 0) v *= theta[j - 1 + s];
                    a[s][nn] = v;
                }
            int ok = oracle_p4_remap(deg, a, M, dM[j], dM[j + 1], out);
            for (int nn = 0; nn <= deg; ++nn) {
                int idx = PPB_FAM[d][f][1 + nn];
                mn[idx][i] = ok ? out[nn] : m[idx][j];
            }
        }
    }
    /* H9, second part: the pressure from the conserved energy with beta of the NEW f (the cell mean just remapped) */
    for (int j = NG; j < nt - NG; ++j) {
        const int i = j - NG;
        const double beta1 = oracle_mix_beta(mn[0][i], gamma1, gamma2);
        const double p1 = fmax(p_floor, (E1[j] - KE1[j]) / beta1);
        qn[4][i] = p1 - p0c[j];
    }
    free(buf);
}

/* NEXT-2 (Fig. 3: "a velocity field is applied ... this is linear advection").
 * PPB-only sweep of one pencil: the hydro state is held fixed and FV is advected by the stored velocity field.
 * [reading R22, DESIGN.md]  The gas is taken as uniform (rho = 1: M_i = dx), the velocity at face i+1/2 is the mean
 * of the two cell values, u_f = (u_i + u_{i+1})/2 (exact for the solid-body rotation of Fig. 3, where the
 * component along a sweep does not vary along it), the mass through the face is dM = dt u_f, and P2-P4 are used
 * unchanged.  u: normal velocity with ghosts (nt = n + 8, odd image sign applied); m: 10 coefficients with ghosts. */
void oracle_advect_pencil(int n, int d, double dx, double dt, const double *u, const double *const m[10],
                          double *const mn[10]) {
    const int nt = n + 2 * NG;
    double *dM = (double *)calloc((size_t)2 * nt + 2, sizeof(double));
    double *theta = dM + nt + 1;
    for (int f = NG; f <= nt - NG; ++f) dM[f] = dt * 0.5 * (u[f - 1] + u[f]);
    for (int j = 3; j <= nt - 4; ++j) {
        double mm[10];
        for (int k = 0; k < 10; ++k) mm[k] = m[k][j];
        theta[j] = oracle_p2_theta(mm);
    }
    for (int j = NG; j < nt - NG; ++j) {
        const int i = j - NG;
        double M[3] = {dx, dx, dx};
        for (int f = 0; f < 6; ++f) {
            const int deg = PPB_FAM[d][f][0];
            double a[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}}, out[3];
            for (int s = 0; s < 3; ++s)
                for (int nn = 0; nn <= deg; ++nn) {
                    int idx = PPB_FAM[d][f][1 + nn];
                    double v = m[idx][j - 1 + s];
                    if (idx != 0) v *= theta[j - 1 + s];
                    a[s][nn] = v;
                }
            int ok = oracle_p4_remap(deg, a, M, dM[j], dM[j + 1], out);
            for (int nn = 0; nn <= deg; ++nn) {
                int idx = PPB_FAM[d][f][1 + nn];
                mn[idx][i] = ok ? out[nn] : m[idx][j];
            }
        }
    }
    free(dM);
}

/* ------------------------------------------------------------------------------------------
 * 3-D driver
 * ---------------------------------------------------------------------------------------- */
static size_t ncell(const oracle_ctx *c) { return (size_t)c->n[0] * c->n[1] * c->n[2]; }
static size_t cidx(const oracle_ctx *c, int i, int j, int k) { return ((size_t)k * c->n[1] + j) * c->n[0] + i; }

oracle_ctx *oracle_create(int nx, int ny, int nz, const int org[3], double dx, double gamma,
                          double rho_floor, double p_floor, int grav_kind, int grav_n, double s0, double ds,
                          const double center[3], const float *g, const float *rho0, const float *p0,
                          const int bc[6]) {
    if (nx < 1 || ny < 1 || nz < 1 || !(dx > 0.0) || !(gamma > 1.0)) return NULL;
    for (int d = 0; d < 3; ++d)
        if ((bc[2 * d] == OR_BC_PERIODIC) != (bc[2 * d + 1] == OR_BC_PERIODIC)) return NULL;
    if (grav_kind != OR_GRAV_NONE && (grav_n < 2 || !g || !rho0 || !p0 || !(ds > 0.0))) return NULL;
    oracle_ctx *c = (oracle_ctx *)calloc(1, sizeof(oracle_ctx));
    c->n[0] = nx; c->n[1] = ny; c->n[2] = nz;
    for (int d = 0; d < 3; ++d) { c->org[d] = org ? org[d] : 0; c->center[d] = center ? center[d] : 0.0; }
    c->dx = dx; c->gamma = gamma; c->rho_floor = rho_floor; c->p_floor = p_floor;
    c->grav_kind = grav_kind; c->grav_n = grav_n; c->s0 = s0; c->ds = ds;
    if (grav_kind != OR_GRAV_NONE) {
        c->g = (double *)malloc(sizeof(double) * grav_n);
        c->rho0 = (double *)malloc(sizeof(double) * grav_n);
        c->p0 = (double *)malloc(sizeof(double) * grav_n);
        for (int k = 0; k < grav_n; ++k) { c->g[k] = g[k]; c->rho0[k] = rho0[k]; c->p0[k] = p0[k]; }
    }
    for (int k = 0; k < 6; ++k) c->bc[k] = bc[k];
    for (int f = 0; f < NF; ++f) {
        c->q[f] = (double *)calloc(ncell(c), sizeof(double));
        c->qn[f] = (double *)calloc(ncell(c), sizeof(double));
    }
    return c;
}

void oracle_destroy(oracle_ctx *c) {
    if (!c) return;
    for (int f = 0; f < NF; ++f) { free(c->q[f]); free(c->qn[f]); }
    free(c->F3);
    free(c->g); free(c->rho0); free(c->p0);
    free(c);
}

static void cell_base(const oracle_ctx *c, int gi, int gj, int gk, double *rho0, double *p0, double gvec[3]) {
    double X[3] = {(gi + 0.5) * c->dx, (gj + 0.5) * c->dx, (gk + 0.5) * c->dx};
    base_at(c, X, rho0, p0, gvec);
}

/* C1: full (rho, ux, uy, uz, p, m000..m011) fp32 -> perturbation form, fp64.  fields[f] = [nz][ny][nx]. */
int oracle_set_state(oracle_ctx *c, const float *const fields[NF]) {
    for (int k = 0; k < c->n[2]; ++k)
        for (int j = 0; j < c->n[1]; ++j)
            for (int i = 0; i < c->n[0]; ++i) {
                size_t id = cidx(c, i, j, k);
                double r0, p0, gv[3];
                cell_base(c, c->org[0] + i, c->org[1] + j, c->org[2] + k, &r0, &p0, gv);
                for (int f = 0; f < NF; ++f) c->q[f][id] = (double)fields[f][id];
                c->q[0][id] -= r0;
                c->q[4][id] -= p0;
            }
    return 0;
}

int oracle_get_state(const oracle_ctx *c, double *const fields[NF]) {
    for (int k = 0; k < c->n[2]; ++k)
        for (int j = 0; j < c->n[1]; ++j)
            for (int i = 0; i < c->n[0]; ++i) {
                size_t id = cidx(c, i, j, k);
                double r0, p0, gv[3];
                cell_base(c, c->org[0] + i, c->org[1] + j, c->org[2] + k, &r0, &p0, gv);
                for (int f = 0; f < NF; ++f) fields[f][id] = c->q[f][id];
                fields[0][id] += r0;
                fields[4][id] += p0;
            }
    return 0;
}

/* raw perturbation-form access (for tests) */
double *oracle_raw_field(oracle_ctx *c, int f) { return c->q[f]; }

/* adiabatic index of a cell: gamma, or Gamma(f) of the two-fluid EOS (NEXT-4, reading R25) with f = its PPB cell mean */
static double cell_gamma(const oracle_ctx *c, size_t id) {
    return c->twofluid ? oracle_mix_gamma(c->q[5][id], c->gamma1, c->gamma2) : c->gamma;
}

/* NEXT-4: switch the two-fluid EOS on (gamma1: the tracked fluid, gamma2: the rest; both > 1) or off */
int oracle_set_two_fluid(oracle_ctx *c, int on, double gamma1, double gamma2) {
    if (!c) return 1;
    if (!on) { c->twofluid = 0; return 0; }
    if (!(gamma1 > 1.0) || !(gamma2 > 1.0) || c->sphere) return 1;     /* (not combined with the confining sphere) */
    c->twofluid = 1; c->gamma1 = gamma1; c->gamma2 = gamma2;
    return 0;
}

static int sweep_impl_sphere(oracle_ctx *c, int d, double dt);   /* NEXT-3, below */
static int cell_is_solid(const oracle_ctx *c, int gi, int gj, int gk);

/* C2/C3/C4/C5: one sweep along d over every pencil of the window. */
static int sweep_impl(oracle_ctx *c, int d, double dt) {
    const int n = c->n[d];
    const int d1 = (d == 0) ? 1 : 0, d2 = (d == 2) ? 1 : 2;   /* transverse axes, ascending */
    const int n1 = c->n[d1], n2 = c->n[d2];
    const int nt = n + 2 * NG;
    /* field index of the normal / transverse velocities for this direction */
    const int iu = 1 + d, iv = 1 + d1, iw = 1 + d2;
    int fail = 0;
#pragma omp parallel for collapse(2) schedule(static)
    for (int b = 0; b < n2; ++b)
        for (int a = 0; a < n1; ++a) {
            double *buf = (double *)malloc(sizeof(double) * ((size_t)nt * 21 + 2 + (size_t)n * 15));
            if (!buf) { fail = 1; continue; }
            double *qa[5], *ma[10], *r0c, *p0c, *gd, *r0f, *p0f, *qo[5], *mo[10];
            double *cur = buf;
            for (int k = 0; k < 5; ++k) { qa[k] = cur; cur += nt; }
            for (int k = 0; k < 10; ++k) { ma[k] = cur; cur += nt; }
            r0c = cur; cur += nt; p0c = cur; cur += nt; gd = cur; cur += nt;
            r0f = cur; cur += nt + 1; p0f = cur; cur += nt + 1;
            double *f3 = cur; cur += nt;
            for (int k = 0; k < 5; ++k) { qo[k] = cur; cur += n; }
            for (int k = 0; k < 10; ++k) { mo[k] = cur; cur += n; }
            int ijk[3], gidx[3];
            ijk[d1] = a; ijk[d2] = b;
            gidx[d1] = c->org[d1] + a; gidx[d2] = c->org[d2] + b;
            for (int j = 0; j < nt; ++j) {
                int sgn, gpos;
                int s = image_cell(c, d, j - NG, &sgn, &gpos);
                ijk[d] = s; gidx[d] = gpos;
                size_t id = cidx(c, ijk[0], ijk[1], ijk[2]);
                qa[0][j] = c->q[0][id];
                qa[1][j] = sgn * c->q[iu][id];
                qa[2][j] = c->q[iv][id];
                qa[3][j] = c->q[iw][id];
                qa[4][j] = c->q[4][id];
                for (int k = 0; k < 10; ++k) ma[k][j] = (ppb_is_odd(d, k) ? sgn : 1) * c->q[5 + k][id];
                double gv[3];
                cell_base(c, gidx[0], gidx[1], gidx[2], &r0c[j], &p0c[j], gv);
                gd[j] = sgn * gv[d];
                f3[j] = (c->flat3d && c->F3) ? c->F3[id] : 0.0;    /* a ghost cell carries its image's F~ (the detector is mirror-invariant) */
            }
            for (int f = 0; f <= nt; ++f) {
                int gf = image_face(c, d, f - NG);
                double X[3], gv[3];
                X[d1] = (gidx[d1] + 0.5) * c->dx; X[d2] = (gidx[d2] + 0.5) * c->dx; X[d] = gf * c->dx;
                base_at(c, X, &r0f[f], &p0f[f], gv);
            }
            if (c->twofluid)
                oracle_sweep_pencil_2f(n, d, c->dx, dt, c->gamma1, c->gamma2, c->rho_floor, c->p_floor,
                                       (const double *const *)qa, (const double *const *)ma, r0c, p0c, gd, r0f, p0f, qo, mo,
                                       (c->flat3d && c->F3) ? f3 : NULL);
            else
            oracle_sweep_pencil(n, d, c->dx, dt, c->gamma, c->rho_floor, c->p_floor,
                                (const double *const *)qa, (const double *const *)ma, r0c, p0c, gd, r0f, p0f, qo, mo,
                                (c->flat3d && c->F3) ? f3 : NULL);
            for (int i = 0; i < n; ++i) {
                ijk[d] = i;
                size_t id = cidx(c, ijk[0], ijk[1], ijk[2]);
                c->qn[0][id] = qo[0][i];
                c->qn[iu][id] = qo[1][i];
                c->qn[iv][id] = qo[2][i];
                c->qn[iw][id] = qo[3][i];
                c->qn[4][id] = qo[4][i];
                for (int k = 0; k < 10; ++k) c->qn[5 + k][id] = mo[k][i];
            }
            free(buf);
        }
    if (fail) return 2;
    for (int f = 0; f < NF; ++f) { double *t = c->q[f]; c->q[f] = c->qn[f]; c->qn[f] = t; }
    return 0;
}

/* NEXT-1 ("a fully 3-D treatment of the shock dissipation ... we evaluate in 3-D the
 * strength and orientation of shocks").  [reading R5b, DESIGN.md]  F~_i = max over the three directions d of the
 * H4 coefficient f~^d_i, each evaluated along d (full p at i-2..i+2, velocity component u_d at i-1, i+1, c_i) on
 * the state the call starts from; ghost cells by the boundary images of C3.  A sweep then spreads it as H4 does:
 * f_i = max(F~_{i-1}, F~_i, F~_{i+1}) along the sweep direction.  So a shock seen in ANY direction flattens the
 * parabolas of EVERY sweep through its cells, which removes the imprint of the grid directions. */
int oracle_set_flatten3d(oracle_ctx *c, int on) {
    if (!c) return 1;
    c->flat3d = on ? 1 : 0;
    if (on && !c->F3) c->F3 = (double *)calloc(ncell(c), sizeof(double));
    return (on && !c->F3) ? 2 : 0;
}

int oracle_flatten3d_update(oracle_ctx *c) {
    if (!c || !c->F3) return 1;
#pragma omp parallel for collapse(2) schedule(static)
    for (int k = 0; k < c->n[2]; ++k)
        for (int j = 0; j < c->n[1]; ++j)
            for (int i = 0; i < c->n[0]; ++i) {
                const int ijk0[3] = {i, j, k};
                double F = 0.0;
                for (int d = 0; d < 3; ++d) {
                    double p5[5], u3[3], ci = 0.0;
                    for (int o = -2; o <= 2; ++o) {
                        int ijk[3] = {ijk0[0], ijk0[1], ijk0[2]}, g[3], sgn, gpos;
                        ijk[d] = image_cell(c, d, ijk0[d] + o, &sgn, &gpos);
                        for (int e = 0; e < 3; ++e) g[e] = c->org[e] + ijk[e];
                        g[d] = gpos;
                        size_t id = cidx(c, ijk[0], ijk[1], ijk[2]);
                        double r0, p0, gv[3];
                        cell_base(c, g[0], g[1], g[2], &r0, &p0, gv);
                        p5[o + 2] = p0 + c->q[4][id];
                        if (o >= -1 && o <= 1) u3[o + 1] = sgn * c->q[1 + d][id];
                        if (o == 0) ci = sqrt(cell_gamma(c, id) * p5[2] / (r0 + c->q[0][id]));
                    }
                    F = fmax(F, oracle_h4_ftilde(p5, u3[0], u3[2], ci));
                }
                c->F3[cidx(c, i, j, k)] = F;
            }
    return 0;
}

const double *oracle_flatten3d_field(const oracle_ctx *c) { return c ? c->F3 : NULL; }

/* one sweep on its own; in 3-D flattening mode F~ is evaluated on the state this sweep starts from */
int oracle_sweep(oracle_ctx *c, int d, double dt) {
    if (!c || d < 0 || d > 2 || !(dt > 0.0)) return 1;
    if (c->sphere) return c->flat3d ? 1 : sweep_impl_sphere(c, d, dt);   /* (the two NEXT modes are not combined) */
    if (c->flat3d) oracle_flatten3d_update(c);
    return sweep_impl(c, d, dt);
}

/* C2: sweep_order 0..5 = xyz, xzy, yxz, yzx, zxy, zyx; one dt for the three sweeps. */
static const int ORDERS[6][3] = {{0, 1, 2}, {0, 2, 1}, {1, 0, 2}, {1, 2, 0}, {2, 0, 1}, {2, 1, 0}};
int oracle_step(oracle_ctx *c, double dt, int sweep_order) {
    if (!c || !(dt > 0.0) || sweep_order < 0 || sweep_order > 5) return 1;
    if (c->sphere && c->flat3d) return 1;
    if (c->flat3d) oracle_flatten3d_update(c);      /* once per step, on the step's starting state */
    for (int s = 0; s < 3; ++s) {
        int rc = c->sphere ? sweep_impl_sphere(c, ORDERS[sweep_order][s], dt) : sweep_impl(c, ORDERS[sweep_order][s], dt);
        if (rc) return rc;
    }
    return 0;
}

/* NEXT-2: PPB-only sweep along d over every pencil; the five hydro fields are not touched. */
static int advect_sweep(oracle_ctx *c, int d, double dt) {
    const int n = c->n[d];
    const int d1 = (d == 0) ? 1 : 0, d2 = (d == 2) ? 1 : 2;
    const int n1 = c->n[d1], n2 = c->n[d2];
    const int nt = n + 2 * NG;
    int fail = 0;
#pragma omp parallel for collapse(2) schedule(static)
    for (int b = 0; b < n2; ++b)
        for (int a = 0; a < n1; ++a) {
            double *buf = (double *)malloc(sizeof(double) * ((size_t)nt * 11 + (size_t)n * 10));
            if (!buf) { fail = 1; continue; }
            double *ua = buf, *ma[10], *mo[10], *cur = buf + nt;
            for (int k = 0; k < 10; ++k) { ma[k] = cur; cur += nt; }
            for (int k = 0; k < 10; ++k) { mo[k] = cur; cur += n; }
            int ijk[3];
            ijk[d1] = a; ijk[d2] = b;
            for (int j = 0; j < nt; ++j) {
                int sgn, gpos;
                ijk[d] = image_cell(c, d, j - NG, &sgn, &gpos);
                size_t id = cidx(c, ijk[0], ijk[1], ijk[2]);
                ua[j] = sgn * c->q[1 + d][id];
                for (int k = 0; k < 10; ++k) ma[k][j] = (ppb_is_odd(d, k) ? sgn : 1) * c->q[5 + k][id];
            }
            oracle_advect_pencil(n, d, c->dx, dt, ua, (const double *const *)ma, mo);
            for (int i = 0; i < n; ++i) {
                ijk[d] = i;
                size_t id = cidx(c, ijk[0], ijk[1], ijk[2]);
                for (int k = 0; k < 10; ++k) c->qn[5 + k][id] = mo[k][i];
            }
            free(buf);
        }
    if (fail) return 2;
    for (int f = 5; f < NF; ++f) { double *t = c->q[f]; c->q[f] = c->qn[f]; c->qn[f] = t; }
    return 0;
}

/* NEXT-2: one PPB-only step = three PPB-only sweeps in the given order with one dt. */
int oracle_advect(oracle_ctx *c, double dt, int sweep_order) {
    if (!c || !(dt > 0.0) || sweep_order < 0 || sweep_order > 5) return 1;
    for (int s = 0; s < 3; ++s) {
        int rc = advect_sweep(c, ORDERS[sweep_order][s], dt);
        if (rc) return rc;
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * NEXT-3: "our star is enclosed in an impenetrable and immovable sphere that is
 * inscribed in the cubical domain of our uniform Cartesian grid ... a very simple boundary condition at the sphere".
 * [reading R23, DESIGN.md]  A cell is SOLID when its centre lies outside the sphere,
 *     ((X - cx)^2 + (Y - cy)^2) + (Z - cz)^2 > R^2      (fp64, each operation rounded, this association),
 * and is never changed.  Along a pencil the fluid cells form one segment [lo, hi] (the sphere is convex); each face
 * between a fluid and a solid cell is a reflecting wall for that sweep: the ghost cells beyond it are the mirror images
 * ALONG THE PENCIL of the segment's own cells (C3: normal velocity and the FV coefficients odd in the normal direction
 * change sign; base state of the mirror-image position, normal g odd), reflected again at the segment's other end when
 * the segment is shorter than the four ghost cells.  So no mass crosses a solid face and a state at rest stays at rest.
 * A segment end that lies on the window boundary keeps the boundary's own rule (REFLECT: the same mirror; OPEN).
 * Reduces to the plain reflecting box when the sphere contains the whole grid.
 * ---------------------------------------------------------------------------------------- */
int oracle_set_sphere(oracle_ctx *c, int on, double radius, const double center[3]) {
    if (!c) return 1;
    if (on) {
        if (!(radius > 0.0) || !center || c->twofluid) return 1;
        for (int d = 0; d < 3; ++d)
            if (c->bc[2 * d] == OR_BC_PERIODIC) return 1;     /* a wall all round: periodic faces make no sense here */
        c->sph_r = radius;
        for (int d = 0; d < 3; ++d) c->sph_c[d] = center[d];
    }
    c->sphere = on ? 1 : 0;
    return 0;
}

/* global cell (gi, gj, gk): 1 if its centre is outside the sphere */
static int cell_is_solid(const oracle_ctx *c, int gi, int gj, int gk) {
    if (!c->sphere) return 0;
    double x = (gi + 0.5) * c->dx - c->sph_c[0], y = (gj + 0.5) * c->dx - c->sph_c[1], z = (gk + 0.5) * c->dx - c->sph_c[2];
    double xx = x * x, yy = y * y, zz = z * z;
    double s = xx + yy;
    s = s + zz;
    return s > c->sph_r * c->sph_r;
}
int oracle_cell_is_solid(const oracle_ctx *c, int i, int j, int k) {
    return cell_is_solid(c, c->org[0] + i, c->org[1] + j, c->org[2] + k);
}

/* image of window-local cell index i along d for a fluid segment [lo, hi] whose ends are walls (lw / hw = 1) or the
 * window's OPEN sides: source index, sign, and the global index whose position supplies the base state */
static int segment_image_cell(const oracle_ctx *c, int d, int lo, int hi, int lw, int hw, int i, int *sgn, int *gpos) {
    int s = i, sg = 1;
    for (int it = 0; it < 64; ++it) {
        if (s < lo) {
            if (!lw) { *sgn = 1; *gpos = c->org[d] + i; return lo; }         /* OPEN: zero gradient, true position */
            s = 2 * lo - 1 - s; sg = -sg;
        } else if (s > hi) {
            if (!hw) { *sgn = 1; *gpos = c->org[d] + i; return hi; }
            s = 2 * hi + 1 - s; sg = -sg;
        } else break;
    }
    *sgn = sg; *gpos = c->org[d] + s;
    return s;
}
/* image of face index f (faces lo .. hi+1 bound the segment) -> global face index */
static int segment_image_face(const oracle_ctx *c, int d, int lo, int hi, int lw, int hw, int f) {
    int s = f;
    for (int it = 0; it < 64; ++it) {
        if (s < lo) { if (!lw) return c->org[d] + f; s = 2 * lo - s; }
        else if (s > hi + 1) { if (!hw) return c->org[d] + f; s = 2 * (hi + 1) - s; }
        else break;
    }
    return c->org[d] + s;
}

/* one sweep along d with the confining sphere: every pencil is cut down to its fluid segment */
static int sweep_impl_sphere(oracle_ctx *c, int d, double dt) {
    const int n = c->n[d];
    const int d1 = (d == 0) ? 1 : 0, d2 = (d == 2) ? 1 : 2;
    const int n1 = c->n[d1], n2 = c->n[d2];
    const int iu = 1 + d, iv = 1 + d1, iw = 1 + d2;
    int fail = 0;
#pragma omp parallel for collapse(2) schedule(static)
    for (int b = 0; b < n2; ++b)
        for (int a = 0; a < n1; ++a) {
            int ijk[3], gidx[3];
            ijk[d1] = a; ijk[d2] = b;
            gidx[d1] = c->org[d1] + a; gidx[d2] = c->org[d2] + b;
            /* the solid cells keep their state */
            for (int i = 0; i < n; ++i) {
                ijk[d] = i;
                size_t id = cidx(c, ijk[0], ijk[1], ijk[2]);
                for (int f = 0; f < NF; ++f) c->qn[f][id] = c->q[f][id];
            }
            int lo = -1, hi = -2;
            for (int i = 0; i < n; ++i) {
                gidx[d] = c->org[d] + i;
                if (!cell_is_solid(c, gidx[0], gidx[1], gidx[2])) { if (lo < 0) lo = i; hi = i; }
            }
            if (lo < 0) continue;                                   /* no fluid on this pencil */
            const int L = hi - lo + 1, nt = L + 2 * NG;
            const int lw = (lo > 0) || c->bc[2 * d] == OR_BC_REFLECT, hw = (hi < n - 1) || c->bc[2 * d + 1] == OR_BC_REFLECT;
            double *buf = (double *)malloc(sizeof(double) * ((size_t)nt * 21 + 2 + (size_t)L * 15));
            if (!buf) { fail = 1; continue; }
            double *qa[5], *ma[10], *r0c, *p0c, *gd, *r0f, *p0f, *qo[5], *mo[10];
            double *cur = buf;
            for (int k = 0; k < 5; ++k) { qa[k] = cur; cur += nt; }
            for (int k = 0; k < 10; ++k) { ma[k] = cur; cur += nt; }
            r0c = cur; cur += nt; p0c = cur; cur += nt; gd = cur; cur += nt;
            r0f = cur; cur += nt + 1; p0f = cur; cur += nt + 1;
            cur += nt;
            for (int k = 0; k < 5; ++k) { qo[k] = cur; cur += L; }
            for (int k = 0; k < 10; ++k) { mo[k] = cur; cur += L; }
            for (int j = 0; j < nt; ++j) {
                int sgn, gpos;
                int s = segment_image_cell(c, d, lo, hi, lw, hw, lo + j - NG, &sgn, &gpos);
                ijk[d] = s; gidx[d] = gpos;
                size_t id = cidx(c, ijk[0], ijk[1], ijk[2]);
                qa[0][j] = c->q[0][id];
                qa[1][j] = sgn * c->q[iu][id];
                qa[2][j] = c->q[iv][id];
                qa[3][j] = c->q[iw][id];
                qa[4][j] = c->q[4][id];
                for (int k = 0; k < 10; ++k) ma[k][j] = (ppb_is_odd(d, k) ? sgn : 1) * c->q[5 + k][id];
                double gv[3];
                cell_base(c, gidx[0], gidx[1], gidx[2], &r0c[j], &p0c[j], gv);
                gd[j] = sgn * gv[d];
            }
            for (int f = 0; f <= nt; ++f) {
                int gf = segment_image_face(c, d, lo, hi, lw, hw, lo + f - NG);
                double X[3], gv[3];
                X[d1] = (gidx[d1] + 0.5) * c->dx; X[d2] = (gidx[d2] + 0.5) * c->dx; X[d] = gf * c->dx;
                base_at(c, X, &r0f[f], &p0f[f], gv);
            }
            oracle_sweep_pencil(L, d, c->dx, dt, c->gamma, c->rho_floor, c->p_floor,
                                (const double *const *)qa, (const double *const *)ma, r0c, p0c, gd, r0f, p0f, qo, mo, NULL);
            for (int i = 0; i < L; ++i) {
                ijk[d] = lo + i;
                size_t id = cidx(c, ijk[0], ijk[1], ijk[2]);
                c->qn[0][id] = qo[0][i];
                c->qn[iu][id] = qo[1][i];
                c->qn[iv][id] = qo[2][i];
                c->qn[iw][id] = qo[3][i];
                c->qn[4][id] = qo[4][i];
                for (int k = 0; k < 10; ++k) c->qn[5 + k][id] = mo[k][i];
            }
            free(buf);
        }
    if (fail) return 2;
    for (int f = 0; f < NF; ++f) { double *t = c->q[f]; c->q[f] = c->qn[f]; c->qn[f] = t; }
    return 0;
}

/* NEXT-3 ("We treat the rotation by adding a solid body rotational flow component to our simulation
 * gradually over the first several thousand time steps").  [reading R24]  One increment of that ramp: every fluid
 * cell gets du = domega e_z x (X - centre), i.e. du_x = -domega (Y - cy), du_y = +domega (X - cx), about the sphere's
 * centre (the gravity centre, else the origin, without a sphere); density and pressure are left as they are.  The
 * caller applies it once per step, domega = Omega_target / N_ramp, for the first N_ramp steps. */
int oracle_spin_up(oracle_ctx *c, double domega) {
    if (!c) return 1;
    const double *cen = c->sphere ? c->sph_c : c->center;
    for (int k = 0; k < c->n[2]; ++k)
        for (int j = 0; j < c->n[1]; ++j)
            for (int i = 0; i < c->n[0]; ++i) {
                if (cell_is_solid(c, c->org[0] + i, c->org[1] + j, c->org[2] + k)) continue;
                size_t id = cidx(c, i, j, k);
                double x = (c->org[0] + i + 0.5) * c->dx - cen[0], y = (c->org[1] + j + 0.5) * c->dx - cen[1];
                c->q[1][id] += -domega * y;
                c->q[2][id] += domega * x;
            }
    return 0;
}

/* C6 */
int oracle_cfl_dt(const oracle_ctx *c, double cfl, double *dt_out) {
    double vmax = 0.0;
    for (int k = 0; k < c->n[2]; ++k)
        for (int j = 0; j < c->n[1]; ++j)
            for (int i = 0; i < c->n[0]; ++i) {
                size_t id = cidx(c, i, j, k);
                double r0, p0, gv[3];
                if (cell_is_solid(c, c->org[0] + i, c->org[1] + j, c->org[2] + k)) continue;     /* NEXT-3: fluid cells only */
                cell_base(c, c->org[0] + i, c->org[1] + j, c->org[2] + k, &r0, &p0, gv);
                double rho = r0 + c->q[0][id], p = p0 + c->q[4][id];
                double cs = sqrt(cell_gamma(c, id) * p / rho);
                for (int d = 0; d < 3; ++d) vmax = fmax(vmax, fabs(c->q[1 + d][id]) + cs);
            }
    *dt_out = cfl * c->dx / vmax;
    return 0;
}

/* C7: mass, mom_x, mom_y, mom_z, total energy, tracked mass */
int oracle_reduce_conserved(const oracle_ctx *c, double out[6]) {
    double acc[6] = {0, 0, 0, 0, 0, 0};
    for (int k = 0; k < c->n[2]; ++k)
        for (int j = 0; j < c->n[1]; ++j)
            for (int i = 0; i < c->n[0]; ++i) {
                size_t id = cidx(c, i, j, k);
                double r0, p0, gv[3];
                if (cell_is_solid(c, c->org[0] + i, c->org[1] + j, c->org[2] + k)) continue;     /* NEXT-3: fluid cells only */
                cell_base(c, c->org[0] + i, c->org[1] + j, c->org[2] + k, &r0, &p0, gv);
                double rho = r0 + c->q[0][id], p = p0 + c->q[4][id];
                double u = c->q[1][id], v = c->q[2][id], w = c->q[3][id];
                acc[0] += rho; acc[1] += rho * u; acc[2] += rho * v; acc[3] += rho * w;
                acc[4] += p / (cell_gamma(c, id) - 1.0) + 0.5 * rho * (u * u + v * v + w * w);
                acc[5] += rho * c->q[5][id];
            }
    double dv = c->dx * c->dx * c->dx;
    for (int k = 0; k < 6; ++k) out[k] = acc[k] * dv;
    return 0;
}

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
