// ppm_sweep.cu — the fused PPM hydro + PPB remap sweep kernel (sm_100a).
//
// One thread owns one grid pencil (pencils are independent within a 1-D pass) and
// marches along the sweep axis with a short sliding window held on chip — the paper's pipelined pencil
// update with a barrel shift (Fig. 7), re-designed for SoA planes: lanes run along
// a transverse axis, so no briquette records, transposes or 16||16 vector splices are needed.
//
// Each iteration n loads plane n and finishes cell n-4 (stencil reach 4, L120).  Per iteration:
//   A  second differences d2_{n-1}
//   B  4th-order face value at (n-2)+1/2                 (H1)
//   C  smoothness S_{n-2} -> omega                       (H3)
//   D  C&W-limited parabola of cell n-2, blended         (H2, H3)
//   E  flattening f~_{n-2}; F  f_{n-3} = max of three    (H4)
//   G  flattened parabola of cell n-3
//   H  characteristic tracing of cell n-3                (H5, H6)
//   I  two-shock Riemann solve at face (n-4)+1/2, fluxes (H7, H8)
//   J  conservative update of cell n-4 in increment form (H9)
//   K  PPB remap of cell n-4 from cells n-5, n-4, n-3    (P1-P4)
//
// fp32 arithmetic.  rho and p are carried as perturbations to the base state; every
// difference of nearly equal numbers is taken between perturbation-sized quantities only ("explicitly
// cancel out all large contributions", L35): the Newton iteration runs on p*' = p* - p0f, the update
// adds increments to rho', p' instead of rebuilding them from E.
#include "ppm_internal.h"

namespace {

// ---- field permutations per sweep direction ----------------------------------------------------
// hydro: normal velocity field and the two transverse ones (ascending axes)
template <int DIR> struct Dir;
template <> struct Dir<0> { static constexpr int U = 1, V = 2, W = 3; };
template <> struct Dir<1> { static constexpr int U = 2, V = 1, W = 3; };
template <> struct Dir<2> { static constexpr int U = 3, V = 1, W = 2; };
// PPB families (P3): local order  a0 a1 a2 | b0 b1 | c0 c1 | d0 e0 f0  -> storage index m[0..9]
__device__ constexpr int PPB_PERM[3][10] = {
    {0, 1, 4, 2, 7, 3, 8, 5, 6, 9},
    {0, 2, 5, 1, 7, 3, 9, 4, 6, 8},
    {0, 3, 6, 1, 8, 2, 9, 4, 5, 7}};
// local indices whose coefficient is odd in the normal direction (C3): a1, b1, c1 = 1, 4, 6

__device__ __forceinline__ float sat(float x) { return __saturatef(x); }
__device__ __forceinline__ float med3(float a, float b, float c) { return fmaxf(fminf(a, b), fminf(fmaxf(a, b), c)); }
__device__ __forceinline__ float rcp(float x) { return __fdividef(1.0f, x); }
__device__ __forceinline__ float fdiv(float a, float b) { return __fdividef(a, b); }

// image of a cell / face index outside [0, n) under the boundary condition (C3)
__device__ __forceinline__ int image_cell(int i, int n, int bc_lo, int bc_hi, float& sgn) {
    sgn = 1.0f;
    if (i >= 0 && i < n) return i;
    const int bc = (i < 0) ? bc_lo : bc_hi;
    if (bc == PPM_BC_PERIODIC) return ((i % n) + n) % n;
    sgn = -1.0f;
    int s = (i < 0) ? (-1 - i) : (2 * n - 1 - i);
    return min(max(s, 0), n - 1);
}
__device__ __forceinline__ int image_face(int f, int n, int bc_lo, int bc_hi) {
    if (f >= 0 && f <= n) return (f == n && bc_hi == PPM_BC_PERIODIC) ? 0 : f;
    const int bc = (f < 0) ? bc_lo : bc_hi;
    if (bc == PPM_BC_PERIODIC) return ((f % n) + n) % n;
    int s = (f < 0) ? -f : 2 * n - f;
    return min(max(s, 0), n);
}

// ---- base state (C1) -----------------------------------------------------------------------------
struct Base { float r0, p0, g; };

__device__ __forceinline__ Base table_at(const SweepParams& P, float s) {
    float t = (s - P.s0) * P.inv_ds;
    int k = (int)floorf(t);
    k = min(max(k, 0), P.tab_n - 2);
    float w = t - (float)k;
    float4 a = __ldg(P.tab + k), b = __ldg(P.tab + k + 1);
    Base o;
    o.g = fmaf(w, b.x - a.x, a.x);
    o.r0 = fmaf(w, b.y - a.y, a.y);
    o.p0 = fmaf(w, b.z - a.z, a.z);
    return o;
}

// per-thread geometry for the base state
template <int DIR, int GRAV> struct Geo {
    float t2;      // RADIAL: squared transverse distance from the centre
    Base cst;      // CONST_Z, DIR != 2: the base state is constant along the pencil
    __device__ __forceinline__ void init(const SweepParams& P, int a, int b) {
        t2 = 0.f; cst.r0 = cst.p0 = cst.g = 0.f;
        if (GRAV == PPM_GRAV_RADIAL) {
            float xa = ((float)a + 0.5f) * P.dx - P.cen_a, xb = ((float)b + 0.5f) * P.dx - P.cen_b;
            t2 = xa * xa + xb * xb;
        } else if (GRAV == PPM_GRAV_CONST_Z && DIR != 2) {
            float4 v = __ldg(P.tab + 2 * b + 2 * PPM_NGHOST + 1);   // b is the z index for x- and y-sweeps
            cst.r0 = v.y; cst.p0 = v.z; cst.g = 0.f;                // no acceleration along x or y
        }
    }
    // cell centre with image index j (sign sgn for the odd normal acceleration)
    __device__ __forceinline__ Base cell(const SweepParams& P, int j, float sgn) const {
        Base o; o.r0 = o.p0 = o.g = 0.f;
        if (GRAV == PPM_GRAV_CONST_Z) {
            if (DIR == 2) { float4 v = __ldg(P.tab + 2 * j + 2 * PPM_NGHOST + 1); o.g = sgn * v.x; o.r0 = v.y; o.p0 = v.z; }
            else o = cst;
        } else if (GRAV == PPM_GRAV_RADIAL) {
            float xd = ((float)j + 0.5f) * P.dx - P.cen_d;
            float r2 = fmaf(xd, xd, t2);
            float ir = rsqrtf(fmaxf(r2, 1e-30f));
            o = table_at(P, r2 * ir);
            o.g = sgn * o.g * xd * ir;
        }
        return o;
    }
    // face with image index f (position f*dx along the sweep axis)
    __device__ __forceinline__ void face(const SweepParams& P, int f, float& r0, float& p0) const {
        r0 = 0.f; p0 = 0.f;
        if (GRAV == PPM_GRAV_CONST_Z) {
            if (DIR == 2) { float4 v = __ldg(P.tab + 2 * f + 2 * PPM_NGHOST); r0 = v.y; p0 = v.z; }
            else { r0 = cst.r0; p0 = cst.p0; }
        } else if (GRAV == PPM_GRAV_RADIAL) {
            float xd = (float)f * P.dx - P.cen_d;
            float r2 = fmaf(xd, xd, t2);
            Base o = table_at(P, sqrtf(r2));
            r0 = o.r0; p0 = o.p0;
        }
    }
};

// ---- H2 + H3: limited parabola blended with the unlimited one ------------------------------------
__device__ __forceinline__ void parabola(float qm, float q0, float qp, float fl, float fr, float om, float& L, float& R) {
    float Lm = med3(qm, fl, q0), Rm = med3(q0, fr, qp);
    const bool ext = (Rm - q0) * (q0 - Lm) <= 0.0f;
    const float D = Rm - Lm, q6 = 6.0f * (q0 - 0.5f * (Lm + Rm));
    const float Dq6 = D * q6, D2 = D * D;
    float L2 = (Dq6 > D2) ? fmaf(-2.0f, Rm, 3.0f * q0) : Lm;
    float R2 = (Dq6 < -D2) ? fmaf(-2.0f, Lm, 3.0f * q0) : Rm;
    Lm = ext ? q0 : L2;
    Rm = ext ? q0 : R2;
    L = fmaf(om, Lm - fl, fl);
    R = fmaf(om, Rm - fr, fr);
}

// ---- H5: A+(s) = qR - F+(q;s),  A-(s) = F-(q;s) - qL ------------------------------------------------
__device__ __forceinline__ float Aplus(float dq, float q6, float s) { return 0.5f * s * (dq - (1.0f - (2.0f / 3.0f) * s) * q6); }
__device__ __forceinline__ float Aminus(float dq, float q6, float s) { return 0.5f * s * (dq + (1.0f - (2.0f / 3.0f) * s) * q6); }

// ---- P4: exact projection of up to three pieces onto the Legendre basis ---------------------------
// S[s][0..9]: pre-limited coefficients (local family order) of cells i-1, i, i+1; rm,r0,rp their masses
// per dx; dl, dr = mass per dx through the left / right face (positive rightward).
__device__ __forceinline__ void ppb_remap(const float (&S)[3][10], float rm, float r0, float rp, float dl, float dr,
                                          float (&out)[10]) {
    const float rn = r0 - dr + dl;
    const bool ok = rn > PPM_TINY;
    const float irn = rcp(fmaxf(rn, PPM_TINY));
    const float dlp = fmaxf(dl, 0.f), dln = fmaxf(-dl, 0.f), drp = fmaxf(dr, 0.f), drn = fmaxf(-dr, 0.f);
    const float irm = rcp(rm), ir0 = rcp(r0), irp = rcp(rp);
    const float w1 = dlp * irn, w3 = drn * irn;          // widths of the donor pieces in the new cell
    // piece geometry: new-coordinate midpoint xm, half width h; old-coordinate midpoint sm, slope beta
    float xm[3], h[3], sm[3], be[3];
    h[0] = 0.5f * w1;              xm[0] = -0.5f + h[0];          sm[0] = 0.5f - 0.5f * dlp * irm;   be[0] = rn * irm;
    h[2] = 0.5f * w3;              xm[2] = 0.5f - h[2];           sm[2] = -0.5f + 0.5f * drn * irp;  be[2] = rn * irp;
    h[1] = 0.5f - h[0] - h[2];     xm[1] = h[0] - h[2];           sm[1] = 0.5f * (dln - drp) * ir0;  be[1] = rn * ir0;
    // reference constants (own cell's degree-0 coefficients): projecting a constant is exact, so only
    // deviations from it are integrated (keeps fp32 round-off at the size of the variation)
    const float refA = S[1][0], refB = S[1][3], refC = S[1][5];
    float a0 = 0.f, a1 = 0.f, a2 = 0.f, b0 = 0.f, b1 = 0.f, c0 = 0.f, c1 = 0.f, d0 = 0.f, e0 = 0.f, f0 = 0.f;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const float hh = h[k], h2 = hh * hh, w = 2.0f * hh;
        const float h23 = h2 * (1.0f / 3.0f), h45 = h2 * h2 * 0.2f;
        const float x = xm[k], x2 = fmaf(x, x, -1.0f / 12.0f);
        const float s = sm[k], s2 = fmaf(s, s, -1.0f / 12.0f), b = be[k];
        const float* c = S[k];
        {   // degree-2 family
            const float E2 = c[2] * b * b, E1 = b * fmaf(2.0f * c[2], s, c[1]);
            const float E0 = (c[0] - refA) + fmaf(c[1], s, c[2] * s2);
            const float J0 = w * fmaf(E2, h23, E0), J1 = w * E1 * h23, J2 = w * fmaf(E0, h23, E2 * h45);
            a0 += J0;
            a1 += fmaf(x, J0, J1);
            a2 += fmaf(x2, J0, fmaf(2.0f * x, J1, J2));
        }
        {   // the two degree-1 families
            const float E0b = (c[3] - refB) + c[4] * s, E1b = b * c[4];
            const float J0b = w * E0b, J1b = w * E1b * h23;
            b0 += J0b; b1 += fmaf(x, J0b, J1b);
            const float E0c = (c[5] - refC) + c[6] * s, E1c = b * c[6];
            const float J0c = w * E0c, J1c = w * E1c * h23;
            c0 += J0c; c1 += fmaf(x, J0c, J1c);
        }
        d0 = fmaf(w, c[7], d0); e0 = fmaf(w, c[8], e0); f0 = fmaf(w, c[9], f0);
    }
    out[0] = ok ? refA + a0 : S[1][0];
    out[1] = ok ? 12.0f * a1 : S[1][1];
    out[2] = ok ? 180.0f * a2 : S[1][2];
    out[3] = ok ? refB + b0 : S[1][3];
    out[4] = ok ? 12.0f * b1 : S[1][4];
    out[5] = ok ? refC + c0 : S[1][5];
    out[6] = ok ? 12.0f * c1 : S[1][6];
    out[7] = ok ? d0 : S[1][7];
    out[8] = ok ? e0 : S[1][8];
    out[9] = ok ? f0 : S[1][9];
}

// ---- the sweep kernel ---------------------------------------------------------------------------------
template <int DIR, int GRAV>
__global__ void __launch_bounds__(128) ppm_sweep_kernel(const SweepParams P) {
    const int a = blockIdx.x * blockDim.x + threadIdx.x;
    if (a >= P.na) return;
    const int b = blockIdx.y;
    const int c0 = blockIdx.z * P.chunk;
    const int c1 = min(c0 + P.chunk, P.n);
    const long long pbase = (long long)a * P.sa + (long long)b * P.sb;
    const float* __restrict__ in = P.in;
    float* __restrict__ out = P.out;
    const long long NC = P.ncell;
    const float gam = P.gamma, gp = 0.5f * (gam + 1.0f), gm = 0.5f * (gam - 1.0f);
    const float dtdx = P.dtdx, hdt = 0.5f * P.dt;

    Geo<DIR, GRAV> geo;
    geo.init(P, a, b);

    // sliding windows (registers).  q[k][s]: cell n-4+s;  k = rho', u, v, w, p'
    float q[5][5], pf[5], rf[6], gw[5];
#pragma unroll
    for (int s = 0; s < 5; ++s) {
#pragma unroll
        for (int k = 0; k < 5; ++k) q[k][s] = 0.f;
        pf[s] = 1.f; gw[s] = 0.f;
    }
#pragma unroll
    for (int s = 0; s < 6; ++s) rf[s] = 1.f;
    float d2a[5], d2b[5], Fc[5], parL[5], parR[5], WLc[5], Fl[5];
#pragma unroll
    for (int k = 0; k < 5; ++k) { d2a[k] = d2b[k] = Fc[k] = parL[k] = parR[k] = WLc[k] = Fl[k] = 0.f; }
    float ft0 = 0.f, ft1 = 0.f, cs = 1.f, r0fc = 0.f, p0fc = 0.f;
    float mw[3][10];
#pragma unroll
    for (int s = 0; s < 3; ++s)
#pragma unroll
        for (int k = 0; k < 10; ++k) mw[s][k] = 0.f;
    if (GRAV == PPM_GRAV_NONE) { r0fc = 0.f; p0fc = 0.f; }

    for (int n = c0 - PPM_NGHOST; n < c1 + PPM_NGHOST; ++n) {
        // ---- shift windows, load plane n -------------------------------------------------------------
#pragma unroll
        for (int s = 0; s < 4; ++s) {
#pragma unroll
            for (int k = 0; k < 5; ++k) q[k][s] = q[k][s + 1];
            pf[s] = pf[s + 1]; gw[s] = gw[s + 1];
        }
#pragma unroll
        for (int s = 0; s < 5; ++s) rf[s] = rf[s + 1];
        {
            float sgn;
            const int j = image_cell(n, P.n, P.bc_lo, P.bc_hi, sgn);
            const long long id = pbase + (long long)j * P.sd;
            q[0][4] = __ldg(in + id);
            q[1][4] = sgn * __ldg(in + Dir<DIR>::U * NC + id);
            q[2][4] = __ldg(in + Dir<DIR>::V * NC + id);
            q[3][4] = __ldg(in + Dir<DIR>::W * NC + id);
            q[4][4] = __ldg(in + 4 * NC + id);
            const Base bs = geo.cell(P, j, sgn);
            rf[5] = bs.r0 + q[0][4];
            pf[4] = bs.p0 + q[4][4];
            gw[4] = bs.g;
        }
        // ---- A, B, C, D: interpolation of cell n-2 ----------------------------------------------------
        float d2n[5], Fn[5], pLn[5], pRn[5];
#pragma unroll
        for (int k = 0; k < 5; ++k) {
            d2n[k] = q[k][4] - 2.0f * q[k][3] + q[k][2];
            Fn[k] = (7.0f / 12.0f) * (q[k][2] + q[k][3]) - (1.0f / 12.0f) * (q[k][1] + q[k][4]);
            const float S = fdiv(fabsf(d2n[k] - d2a[k]), fabsf(d2a[k]) + 2.0f * fabsf(d2b[k]) + fabsf(d2n[k]) + PPM_TINY);
            const float om = sat((S - 0.1f) * 5.0f);
            parabola(q[k][1], q[k][2], q[k][3], Fc[k], Fn[k], om, pLn[k], pRn[k]);
        }
        // ---- E, F: flattening ---------------------------------------------------------------------------
        const float cn2 = sqrtf(gam * pf[2] * rcp(rf[3]));          // c_{n-2}
        float ftn;
        {
            const float d1 = pf[3] - pf[1], dd2 = pf[4] - pf[0];
            const float steep = sat(10.0f * (fdiv(fabsf(d1), fmaxf(fabsf(dd2), PPM_TINY)) - 0.75f));
            const float jump = sat(fdiv(3.0f * fabsf(d1), fminf(pf[3], pf[1])) - 1.0f);
            const float conv = sat(fdiv(q[1][1] - q[1][3], 0.05f * cn2));
            ftn = steep * jump * conv;
        }
        const float fl3 = fmaxf(ft0, fmaxf(ft1, ftn));              // f_{n-3}
        // ---- G, H: flattened parabola and characteristic tracing of cell n-3 ---------------------------
        float WL[5], WR[5];
        float r0fn, p0fn;
        {
            const int fi = image_face(n - 2, P.n, P.bc_lo, P.bc_hi);
            geo.face(P, fi, r0fn, p0fn);
        }
        {
            float qL[5], dq[5], q6[5];
#pragma unroll
            for (int k = 0; k < 5; ++k) {
                const float qc = q[k][1];
                const float L = fmaf(fl3, qc - parL[k], parL[k]);
                const float R = fmaf(fl3, qc - parR[k], parR[k]);
                qL[k] = L; dq[k] = R - L; q6[k] = 6.0f * (qc - 0.5f * (L + R));
            }
            const float rho = rf[2], c = cs, u = q[1][1];
            const float rc = rho * c, ic2h = 0.5f * rcp(c * c), cor = fdiv(c, rho);   // 1/(2c^2), c/rho
            const float s_m = (u - c) * dtdx, s_0 = u * dtdx, s_p = (u + c) * dtdx;
            // Each wave family k takes its amplitude from its own domain of dependence max(+-sigma^k, 0); a
            // wave moving away from the face has the zero-width domain, i.e. the edge value (reading R8',
            // DESIGN.md).  No switch on sign(lambda^k): the traced states are continuous in the data.
            // left of face (n-3)+1/2 : W~ = qR - A+(max(s_p,0));  delta^k = W~ - F+(s_k) = A+(s_k) - A+(sp)
            {
                const float sp = fmaxf(s_p, 0.f), smk = fmaxf(s_m, 0.f), s0k = fmaxf(s_0, 0.f);
                const float Ar = Aplus(dq[0], q6[0], sp), Au = Aplus(dq[1], q6[1], sp), Ap = Aplus(dq[4], q6[4], sp);
                const float du_m = Aplus(dq[1], q6[1], smk) - Au, dp_m = Aplus(dq[4], q6[4], smk) - Ap;
                const float am = (dp_m - rc * du_m) * ic2h;
                const float dr_0 = Aplus(dq[0], q6[0], s0k) - Ar, dp_0 = Aplus(dq[4], q6[4], s0k) - Ap;
                const float a0 = dr_0 - dp_0 * (2.0f * ic2h);
                const float R0 = qL[0] + dq[0], R1 = qL[1] + dq[1], R4 = qL[4] + dq[4];
                WL[0] = R0 - Ar - am - a0;
                WL[1] = R1 - Au + cor * am;
                WL[4] = R4 - Ap - c * c * am;
                WL[2] = qL[2] + dq[2] - Aplus(dq[2], q6[2], s0k);
                WL[3] = qL[3] + dq[3] - Aplus(dq[3], q6[3], s0k);
            }
            // right of face (n-3)-1/2 : W~ = qL + A-(max(-s_m,0));  delta^k = A-(sm) - A-(max(-s_k,0))
            {
                const float sm = fmaxf(-s_m, 0.f), spk = fmaxf(-s_p, 0.f), s0k = fmaxf(-s_0, 0.f);
                const float Ar = Aminus(dq[0], q6[0], sm), Au = Aminus(dq[1], q6[1], sm), Ap = Aminus(dq[4], q6[4], sm);
                const float du_p = Au - Aminus(dq[1], q6[1], spk), dp_p = Ap - Aminus(dq[4], q6[4], spk);
                const float ap = (dp_p + rc * du_p) * ic2h;
                const float dr_0 = Ar - Aminus(dq[0], q6[0], s0k), dp_0 = Ap - Aminus(dq[4], q6[4], s0k);
                const float a0 = dr_0 - dp_0 * (2.0f * ic2h);
                WR[0] = qL[0] + Ar - ap - a0;
                WR[1] = qL[1] + Au - cor * ap;
                WR[4] = qL[4] + Ap - c * c * ap;
                WR[2] = qL[2] + Aminus(dq[2], q6[2], s0k);
                WR[3] = qL[3] + Aminus(dq[3], q6[3], s0k);
            }
            if (GRAV != PPM_GRAV_NONE) {   // half-step sources of the perturbation equations (H6)
                const float sr = hdt * (-u * (r0fn - r0fc) * P.inv_dx);
                const float sp_ = hdt * (-u * (p0fn - p0fc) * P.inv_dx);
                const float su = hdt * gw[1] * fdiv(q[0][1], rho);
                WL[0] += sr; WR[0] += sr; WL[4] += sp_; WR[4] += sp_; WL[1] += su; WR[1] += su;
            }
        }
        // ---- I: Riemann problem at face (n-4)+1/2 : L = WLc (cell n-4), R = WR (cell n-3) -------------
        float Fr[5];
        {
            const float rL = fmaxf(r0fc + WLc[0], P.rho_floor), rR = fmaxf(r0fc + WR[0], P.rho_floor);
            const float ppL = fmaxf(WLc[4], P.p_floor - p0fc), ppR = fmaxf(WR[4], P.p_floor - p0fc);   // p' (floored)
            const float pL = p0fc + ppL, pR = p0fc + ppR;
            const float uL = WLc[1], uR = WR[1];
            const float CL2 = gam * pL * rL, CR2 = gam * pR * rR;
            const float CL = sqrtf(CL2), CR = sqrtf(CR2);
            const float pfl = P.p_floor - p0fc;
            float pps = fmaxf(pfl, fdiv(CR * ppL + CL * ppR + CL * CR * (uL - uR), CL + CR));             // p*' acoustic guess
            float WLs, WRs;
#pragma unroll
            for (int it = 0; it < 5; ++it) {
                const float ps = p0fc + pps;
                const float wl2 = rL * fmaf(gp, ps, gm * pL), wr2 = rR * fmaf(gp, ps, gm * pR);
                const float iwl = rsqrtf(wl2), iwr = rsqrtf(wr2);
                WLs = wl2 * iwl; WRs = wr2 * iwr;
                const float usl = uL - (pps - ppL) * iwl, usr = uR + (pps - ppR) * iwr;
                const float ZL = fdiv(2.0f * wl2 * WLs, wl2 + CL2), ZR = fdiv(2.0f * wr2 * WRs, wr2 + CR2);
                pps = fmaxf(pfl, pps - fdiv(ZL * ZR * (usr - usl), ZL + ZR));
            }
            const float ps = p0fc + pps;
            const float wl2 = rL * fmaf(gp, ps, gm * pL), wr2 = rR * fmaf(gp, ps, gm * pR);
            WLs = sqrtf(wl2); WRs = sqrtf(wr2);
            const float us = fdiv(WLs * uL + WRs * uR + (ppL - ppR), WLs + WRs);
            // sampling at x/t = 0 in the frame mirrored so that the upwind side K is on the left
            const bool left = us >= 0.f;
            const float sg = left ? 1.f : -1.f;
            const float rK = left ? rL : rR, uK = left ? uL : uR, pK = left ? pL : pR, ppK = left ? ppL : ppR;
            const float wk2 = left ? wl2 : wr2, WK = left ? WLs : WRs;
            const float vK = left ? WLc[2] : WR[2], wK = left ? WLc[3] : WR[3];
            float rs = fdiv(rK * wk2, wk2 - rK * (pps - ppK));                 // 1/(1/rK - (p*-pK)/WK^2)
            rs = fmaxf(rs, P.rho_floor);
            const float cK = sqrtf(gam * pK * rcp(rK)), cst = sqrtf(gam * ps * rcp(rs));
            const float uKh = sg * uK, ush = sg * us;
            const bool shock = pps > ppK;
            const float lam_head = shock ? uKh - fdiv(WK, rK) : uKh - cK;
            const float lam_tail = shock ? lam_head : ush - cst;
            float th = (lam_head >= 0.f) ? 0.f : ((lam_tail <= 0.f) ? 1.f : fdiv(-lam_head, lam_tail - lam_head));
            const float rh = fmaf(th, rs - rK, rK);
            const float uh = fmaf(th, us - uK, uK);
            const float pph = fmaf(th, pps - ppK, ppK);
            const float ph = p0fc + pph;
            const float Fm = rh * uh;
            Fr[0] = Fm;
            Fr[1] = fmaf(Fm, uh, pph);
            Fr[2] = Fm * vK;
            Fr[3] = Fm * wK;
            Fr[4] = uh * fmaf(gam * rcp(gam - 1.0f), ph, 0.5f * rh * (uh * uh + vK * vK + wK * wK));
        }
        // ---- K (first half): PPB coefficients of cell n-3, pre-limited (P2) ---------------------------
#pragma unroll
        for (int k = 0; k < 10; ++k) { mw[0][k] = mw[1][k]; mw[1][k] = mw[2][k]; }
        if (n - 3 >= c0 - 1) {
            float sgn;
            const int j = image_cell(n - 3, P.n, P.bc_lo, P.bc_hi, sgn);
            const long long id = pbase + (long long)j * P.sd;
            float m[10];
#pragma unroll
            for (int k = 0; k < 10; ++k) m[k] = __ldg(in + (long long)(5 + PPB_PERM[DIR][k]) * NC + id);
            m[1] *= sgn; m[4] *= sgn; m[6] *= sgn;
            // storage-order roles for the bound B: first-order terms 1/2, pure second-order 1/6, mixed 1/4.
            // local order: a1,b0,c0 are P1 terms; a2,d0,e0 are P2 terms; b1,c1,f0 are mixed P1P1 terms.
            const float B = 0.5f * (fabsf(m[1]) + fabsf(m[3]) + fabsf(m[5])) + (1.0f / 6.0f) * (fabsf(m[2]) + fabsf(m[7]) + fabsf(m[8]))
                          + 0.25f * (fabsf(m[4]) + fabsf(m[6]) + fabsf(m[9]));
            const float th = fminf(1.0f, fdiv(fmaxf(0.f, fminf(m[0], 1.0f - m[0])), fmaxf(B, PPM_TINY)));
            mw[2][0] = m[0];
#pragma unroll
            for (int k = 1; k < 10; ++k) mw[2][k] = m[k] * th;
        }
        // ---- J, K, L: finish cell n-4 ---------------------------------------------------------------------
        const int i = n - PPM_NGHOST;
        if (i >= c0) {
            const float r_old = rf[1], rp_old = q[0][0], u0 = q[1][0], v0 = q[2][0], w0 = q[3][0], g = gw[0];
            float drho = -dtdx * (Fr[0] - Fl[0]);
            int bad = 0;
            if (!(r_old + drho > P.rho_floor)) { drho = P.rho_floor - r_old; bad = 1; }
            const float r_new = r_old + drho;
            const float rp_new = rp_old + drho;
            const float mu0 = r_old * u0;
            float mu1 = mu0 - dtdx * (Fr[1] - Fl[1]);
            float dE = -dtdx * (Fr[4] - Fl[4]);
            if (GRAV != PPM_GRAV_NONE) {
                mu1 += P.dt * 0.5f * (rp_old + rp_new) * g;
                dE += P.dt * 0.5f * (mu0 + mu1) * g;
            }
            const float mv1 = r_old * v0 - dtdx * (Fr[2] - Fl[2]);
            const float mw1 = r_old * w0 - dtdx * (Fr[3] - Fl[3]);
            const float irn = rcp(r_new);
            const float u1 = mu1 * irn, v1 = mv1 * irn, w1 = mw1 * irn;
            const float dKE = 0.5f * (r_new * (u1 * u1 + v1 * v1 + w1 * w1) - r_old * (u0 * u0 + v0 * v0 + w0 * w0));
            float pp_new = q[4][0] + (gam - 1.0f) * (dE - dKE);
            const float p0c = pf[0] - q[4][0];
            if (!(p0c + pp_new > P.p_floor)) { pp_new = P.p_floor - p0c; bad = 1; }
            if (bad) atomicOr(P.flag, (r_new == r_new && pp_new == pp_new) ? 1 : 2);
            const long long id = pbase + (long long)i * P.sd;
            out[id] = rp_new;
            out[Dir<DIR>::U * NC + id] = u1;
            out[Dir<DIR>::V * NC + id] = v1;
            out[Dir<DIR>::W * NC + id] = w1;
            out[4 * NC + id] = pp_new;
            float mo[10];
            ppb_remap(mw, rf[0], rf[1], rf[2], dtdx * Fl[0], dtdx * Fr[0], mo);
#pragma unroll
            for (int k = 0; k < 10; ++k) out[(long long)(5 + PPB_PERM[DIR][k]) * NC + id] = mo[k];
        }
        // ---- rotate the carried pipeline registers ----------------------------------------------------
#pragma unroll
        for (int k = 0; k < 5; ++k) {
            d2a[k] = d2b[k]; d2b[k] = d2n[k]; Fc[k] = Fn[k]; parL[k] = pLn[k]; parR[k] = pRn[k];
            WLc[k] = WL[k]; Fl[k] = Fr[k];
        }
        ft0 = ft1; ft1 = ftn; cs = cn2; r0fc = r0fn; p0fc = p0fn;
    }
}

template <int DIR>
cudaError_t launch_dir(const SweepParams& P, int grav, dim3 grid, dim3 block, cudaStream_t st) {
    switch (grav) {
        case PPM_GRAV_NONE: ppm_sweep_kernel<DIR, PPM_GRAV_NONE><<<grid, block, 0, st>>>(P); break;
        case PPM_GRAV_CONST_Z: ppm_sweep_kernel<DIR, PPM_GRAV_CONST_Z><<<grid, block, 0, st>>>(P); break;
        default: ppm_sweep_kernel<DIR, PPM_GRAV_RADIAL><<<grid, block, 0, st>>>(P); break;
    }
    return cudaGetLastError();
}

}  // namespace

cudaError_t ppm_launch_sweep(ppm_ctx* c, int axis, double dt) {
    const ppm_params& p = c->prm;
    const long long nx = p.nx, ny = p.ny, nz = p.nz;
    SweepParams P;
    P.in = c->buf[c->cur];
    P.out = c->buf[c->cur ^ 1];
    P.ncell = nx * ny * nz;
    const long long str[3] = {1, nx, nx * ny};
    const int ext[3] = {p.nx, p.ny, p.nz};
    const int ia = (axis == 0) ? 1 : 0;       // thread-mapped transverse axis
    const int ib = (axis == 2) ? 1 : 2;       // blockIdx.y transverse axis
    P.n = ext[axis]; P.na = ext[ia]; P.nb = ext[ib];
    P.sd = str[axis]; P.sa = str[ia]; P.sb = str[ib];
    P.bc_lo = p.bc[2 * axis]; P.bc_hi = p.bc[2 * axis + 1];
    int chunk = c->chunk > 0 ? c->chunk : P.n;
    if (chunk > P.n) chunk = P.n;
    P.chunk = chunk;
    P.dt = (float)dt; P.dx = (float)p.dx; P.dtdx = (float)(dt / p.dx); P.inv_dx = (float)(1.0 / p.dx);
    P.gamma = (float)p.gamma; P.rho_floor = (float)p.rho_floor; P.p_floor = (float)p.p_floor;
    P.tab_n = p.grav.n; P.s0 = (float)p.grav.s0; P.inv_ds = (float)(p.grav.kind != PPM_GRAV_NONE ? 1.0 / p.grav.ds : 0.0);
    P.cen_d = (float)p.grav.center[axis]; P.cen_a = (float)p.grav.center[ia]; P.cen_b = (float)p.grav.center[ib];
    P.tab = c->tab;
    P.flag = c->flag;
    const int nchunks = (P.n + chunk - 1) / chunk;
    dim3 block(128, 1, 1), grid((P.na + 127) / 128, P.nb, nchunks);
    cudaError_t e;
    if (axis == 0) e = launch_dir<0>(P, p.grav.kind, grid, block, c->stream);
    else if (axis == 1) e = launch_dir<1>(P, p.grav.kind, grid, block, c->stream);
    else e = launch_dir<2>(P, p.grav.kind, grid, block, c->stream);
    if (e == cudaSuccess) { c->cur ^= 1; c->launches += 1; }
    return e;
}
