// ppm_sweep.cu — the fused PPM hydro + PPB remap sweep kernels (sm_100a).
//
// One thread owns one grid pencil (pencils are independent within a 1-D pass) and
// marches along the sweep axis with a short sliding window held on chip — the paper's pipelined pencil
// update with a barrel shift (Fig. 7), re-designed for SoA planes: lanes run along
// a transverse axis, so no briquette records, transposes or 16||16 vector splices are needed.
//
// Each iteration n takes plane n and finishes cell n-4 (stencil reach 4, L120).  Per iteration:
//   A  second differences d2_{n-1}
//   B  4th-order face value at (n-2)+1/2, and its clamp  (H1; H2)
//   C  smoothness S_{n-2} -> omega                       (H3)
//   D  C&W-limited parabola of cell n-2, blended         (H2, H3)
//   E  flattening f~_{n-2}; F  f_{n-3} = max of three    (H4)
//   G  flattened parabola of cell n-3
//   H  characteristic tracing of cell n-3                (H5, H6 with reading R8')
//   I  two-shock Riemann solve at face (n-4)+1/2, fluxes (H7, H8)
//   J  conservative update of cell n-4 in increment form (H9)
//   K  PPB remap of cell n-4 from cells n-5, n-4, n-3    (P1-P4)
//
// State layout in HBM: SoA bricks — per field, bricks of 4x4x4 cells (256 B, x fastest inside), bricks
// ordered x-fastest.  Every sweep direction then reads and writes whole 256-byte bricks (measured on SoA
// planes: the x sweep re-read DRAM 6.5x because 16-byte row pieces thrash L2; profiles/).  The paper's
// briquettes answer the same problem; here they are per-field (SoA), so a warp's 32
// pencils = 2 bricks x (4x4 transverse cells) and no on-chip transposition is ever needed.
//
// Two data paths feed the same marching body:
//   IoDirect  y/z sweeps (and grids whose extents are not multiples of 4, kept as SoA planes): loads and
//             stores straight from/to HBM, 16 lanes per brick layer, L1 keeps a brick for the 2-4 iterations
//             that consume it; next plane software-prefetched into registers.
//   IoTmaX    x sweep: each warp stages one brick column step (2 bricks x 5 fields = 2560 B per TMA box,
//             cp.async.bulk.tensor 5-D) into THREAD-PRIVATE 16-byte slots, double buffered behind the
//             arithmetic, and writes results back with TMA stores; no transposes, no bank conflicts.
//
// fp32 arithmetic.  rho and p are carried as perturbations to the base state; every
// difference of nearly equal numbers is taken between perturbation-sized quantities only ("explicitly
// cancel out all large contributions", L35): the Newton iteration runs on p*' = p* - p0f, the update
// adds increments to rho', p' instead of rebuilding them from E.
#include <cuda.h>
#include <stdlib.h>

#include "ppm_internal.h"

#ifndef PPM_MARCH_UNROLL
#define PPM_MARCH_UNROLL 1
#endif

namespace {

constexpr int MARCH_UNROLL = PPM_MARCH_UNROLL;   // iterations of the marching loop per loop body

// ---- field permutations per sweep direction ----------------------------------------------------
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
__device__ __forceinline__ float fsqrt(float x) { return x * rsqrtf(fmaxf(x, 1e-37f)); }

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
            Base o = table_at(P, fsqrt(r2));
            r0 = o.r0; p0 = o.p0;
        }
    }
};

// ---- H2 + H3: limited parabola blended with the unlimited one ------------------------------------
// Lc, Rc: face values already clamped between the neighbouring cell means (per-face medians)
__device__ __forceinline__ void parabola(float q0, float Lc, float Rc, float fl, float fr, float om, float& L, float& R) {
    const bool ext = (Rc - q0) * (q0 - Lc) <= 0.0f;
    const float D = Rc - Lc, q6 = 6.0f * (q0 - 0.5f * (Lc + Rc));
    const float Dq6 = D * q6, D2 = D * D;
    float L2 = (Dq6 > D2) ? fmaf(-2.0f, Rc, 3.0f * q0) : Lc;
    float R2 = (Dq6 < -D2) ? fmaf(-2.0f, Lc, 3.0f * q0) : Rc;
    L2 = ext ? q0 : L2;
    R2 = ext ? q0 : R2;
    L = fmaf(om, L2 - fl, fl);
    R = fmaf(om, R2 - fr, fr);
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

// =====================================================================================================
// The marching body, shared by every data path.  IO supplies plane n (hydro), cell n-3 (PPB coefficients,
// local family order, mirror signs applied) and takes the finished cell n-4.
// =====================================================================================================
template <int DIR, int GRAV, class IO>
__device__ __forceinline__ void march(const SweepParams& P, IO& io, const int a, const int b, const int c0, const int c1,
                                      const bool valid, const unsigned wmask) {
    const float gam = P.gamma, gp = 0.5f * (gam + 1.0f), gm = 0.5f * (gam - 1.0f), g_gm1 = gam * rcp(gam - 1.0f);
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
    float d2a[5], d2b[5], Fc[5], Fcl[5], parL[5], parR[5], WLc[5], Fl[5];
#pragma unroll
    for (int k = 0; k < 5; ++k) { d2a[k] = d2b[k] = Fc[k] = Fcl[k] = parL[k] = parR[k] = WLc[k] = Fl[k] = 0.f; }
    float ft0 = 0.f, ft1 = 0.f, cs = 1.f, r0fc = 0.f, p0fc = 0.f;
    float mw[3][10];
#pragma unroll
    for (int s = 0; s < 3; ++s)
#pragma unroll
        for (int k = 0; k < 10; ++k) mw[s][k] = 0.f;

#pragma unroll MARCH_UNROLL
    for (int n = c0 - PPM_NGHOST; n < c1 + PPM_NGHOST; ++n) {
        io.begin(n);
        // ---- shift windows, take plane n ---------------------------------------------------------------
#pragma unroll
        for (int s = 0; s < 4; ++s) {
#pragma unroll
            for (int k = 0; k < 5; ++k) q[k][s] = q[k][s + 1];
            pf[s] = pf[s + 1]; gw[s] = gw[s + 1];
        }
#pragma unroll
        for (int s = 0; s < 5; ++s) rf[s] = rf[s + 1];
        {
            float sgn, v[5];
            int j;
            io.hydro(n, j, sgn, v);
#pragma unroll
            for (int k = 0; k < 5; ++k) q[k][4] = v[k];
            const Base bs = geo.cell(P, j, sgn);
            rf[5] = bs.r0 + q[0][4];
            pf[4] = bs.p0 + q[4][4];
            gw[4] = bs.g;
        }
        // ---- A, B, C, D: interpolation of cell n-2 ----------------------------------------------------
        float d2n[5], Fn[5], Fnl[5], pLn[5], pRn[5];
#pragma unroll
        for (int k = 0; k < 5; ++k) {
            d2n[k] = q[k][4] - 2.0f * q[k][3] + q[k][2];
            Fn[k] = (7.0f / 12.0f) * (q[k][2] + q[k][3]) - (1.0f / 12.0f) * (q[k][1] + q[k][4]);
            Fnl[k] = med3(q[k][2], Fn[k], q[k][3]);                      // H2: clamp between the adjacent means
            const float S = fdiv(fabsf(d2n[k] - d2a[k]), fabsf(d2a[k]) + 2.0f * fabsf(d2b[k]) + fabsf(d2n[k]) + PPM_TINY);
            const float om = sat((S - 0.1f) * 5.0f);
            parabola(q[k][2], Fcl[k], Fnl[k], Fc[k], Fn[k], om, pLn[k], pRn[k]);
        }
        // ---- E, F: flattening ---------------------------------------------------------------------------
        const float cn2 = fsqrt(gam * pf[2] * rcp(rf[3]));          // c_{n-2}
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
            const float pfl = P.p_floor - p0fc;
            const float ppL = fmaxf(WLc[4], pfl), ppR = fmaxf(WR[4], pfl);           // p' (floored)
            const float pL = p0fc + ppL, pR = p0fc + ppR;
            const float uL = WLc[1], uR = WR[1];
            const float CL2 = gam * pL * rL, CR2 = gam * pR * rR;
            const float CL = fsqrt(CL2), CR = fsqrt(CR2);
            float pps = fmaxf(pfl, fdiv(CR * ppL + CL * ppR + CL * CR * (uL - uR), CL + CR));   // p*' acoustic guess
            const float gpL = gp * rL, gpR = gp * rR, gmL = gm * pL * rL, gmR = gm * pR * rR;
            // Newton on p*' with the two-shock wave speeds W_K; at most 5 iterations (reading R7).  The loop
            // stops early only when EVERY lane's last update is below fp32 resolution of p* (warp-uniform
            // exit), i.e. when further iterations could not change the result beyond rounding.
            auto newton = [&]() -> bool {
                const float ps = p0fc + pps;
                const float wl2 = fmaf(gpL, ps, gmL), wr2 = fmaf(gpR, ps, gmR);
                const float iwl = rsqrtf(wl2), iwr = rsqrtf(wr2);
                const float usl = uL - (pps - ppL) * iwl, usr = uR + (pps - ppR) * iwr;
                // 1/Z_K = (W^2 + C^2) / (2 W^3)
                const float izl = (wl2 + CL2) * (iwl * iwl * iwl), izr = (wr2 + CR2) * (iwr * iwr * iwr);
                const float d = fdiv(2.0f * (usr - usl), izl + izr);
                pps = fmaxf(pfl, pps - d);
                return fabsf(d) <= 6e-8f * ps;
            };
            // first iteration in straight-line code (the scheduler can overlap it with independent work); the
            // remaining ones only while some lane still moves (rare at low Mach: the acoustic guess is nearly exact)
            if (!__all_sync(wmask, newton())) {
#pragma unroll 1
                for (int it = 1; it < 5; ++it)
                    if (__all_sync(wmask, newton())) break;
            }
            const float ps = p0fc + pps;
            const float wl2 = fmaf(gpL, ps, gmL), wr2 = fmaf(gpR, ps, gmR);
            const float WLs = fsqrt(wl2), WRs = fsqrt(wr2);
            const float us = fdiv(WLs * uL + WRs * uR + (ppL - ppR), WLs + WRs);
            // sampling at x/t = 0 in the frame mirrored so that the upwind side K is on the left
            const bool left = us >= 0.f;
            const float sg = left ? 1.f : -1.f;
            const float rK = left ? rL : rR, uK = left ? uL : uR, pK = left ? pL : pR, ppK = left ? ppL : ppR;
            const float wk2 = left ? wl2 : wr2, WK = left ? WLs : WRs;
            const float vK = left ? WLc[2] : WR[2], wK = left ? WLc[3] : WR[3];
            float rs = fdiv(rK * wk2, wk2 - rK * (pps - ppK));                 // 1/(1/rK - (p*-pK)/WK^2)
            rs = fmaxf(rs, P.rho_floor);
            const float irK = rcp(rK);
            const float cK = fsqrt(gam * pK * irK), cst = fsqrt(gam * ps * rcp(rs));
            const float uKh = sg * uK, ush = sg * us;
            const bool shock = pps > ppK;
            const float lam_head = uKh - (shock ? WK * irK : cK);
            const float lam_tail = shock ? lam_head : ush - cst;
            const float th = (lam_head >= 0.f) ? 0.f : ((lam_tail <= 0.f) ? 1.f : fdiv(-lam_head, lam_tail - lam_head));
            const float rh = fmaf(th, rs - rK, rK);
            const float uh = fmaf(th, us - uK, uK);
            const float pph = fmaf(th, pps - ppK, ppK);
            const float ph = p0fc + pph;
            const float Fm = rh * uh;
            Fr[0] = Fm;
            Fr[1] = fmaf(Fm, uh, pph);
            Fr[2] = Fm * vK;
            Fr[3] = Fm * wK;
            Fr[4] = uh * fmaf(g_gm1, ph, 0.5f * rh * (uh * uh + vK * vK + wK * wK));
        }
        // ---- K (first half): PPB coefficients of cell n-3, pre-limited (P2) ---------------------------
#pragma unroll
        for (int k = 0; k < 10; ++k) { mw[0][k] = mw[1][k]; mw[1][k] = mw[2][k]; }
        if (n - 3 >= c0 - 1) {
            float m[10];
            io.ppb(n - 3, m);
            // bound B: first-order terms 1/2, pure second-order 1/6, mixed 1/4.
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
            float ho[5], mo[10];
            const float u1 = mu1 * irn, v1 = mv1 * irn, w1 = mw1 * irn;
            const float dKE = 0.5f * (r_new * (u1 * u1 + v1 * v1 + w1 * w1) - r_old * (u0 * u0 + v0 * v0 + w0 * w0));
            float pp_new = q[4][0] + (gam - 1.0f) * (dE - dKE);
            const float p0c = pf[0] - q[4][0];
            if (!(p0c + pp_new > P.p_floor)) { pp_new = P.p_floor - p0c; bad = 1; }
            if (bad && valid) atomicOr(P.flag, (r_new == r_new && pp_new == pp_new) ? 1 : 2);
            ho[0] = rp_new; ho[1] = u1; ho[2] = v1; ho[3] = w1; ho[4] = pp_new;
            ppb_remap(mw, rf[0], rf[1], rf[2], dtdx * Fl[0], dtdx * Fr[0], mo);
            io.store(i, ho, mo);
        }
        // ---- rotate the carried pipeline registers ----------------------------------------------------
#pragma unroll
        for (int k = 0; k < 5; ++k) {
            d2a[k] = d2b[k]; d2b[k] = d2n[k]; Fc[k] = Fn[k]; Fcl[k] = Fnl[k]; parL[k] = pLn[k]; parR[k] = pRn[k];
            WLc[k] = WL[k]; Fl[k] = Fr[k];
        }
        ft0 = ft1; ft1 = ftn; cs = cn2; r0fc = r0fn; p0fc = p0fn;
        io.end(n);
    }
    io.finish();
}

// =====================================================================================================
// IoDirect: straight global loads / stores, lanes along a contiguous axis; next plane prefetched.
// =====================================================================================================
__device__ __forceinline__ unsigned axis_off(const SweepParams& P, int j) { return (unsigned)(j >> 2) * (unsigned)P.SBd + (unsigned)(j & 3) * (unsigned)P.SId; }

template <int DIR>
struct IoDirect {
    const SweepParams& P;
    const unsigned pbase;    // element offsets inside one field fit 32 bits (ppm_create checks)
    float nx5[5];            // plane n+1, already in flight
    float nm[10];            // PPB coefficients of the next cell, already in flight
    int jn; float sn, snm;
    __device__ __forceinline__ IoDirect(const SweepParams& P_, unsigned pb, int n0, int c0) : P(P_), pbase(pb) { fetch(n0); fetch_ppb(c0 - 1); }
    __device__ __forceinline__ void fetch(int n) {
        jn = image_cell(n, P.n, P.bc_lo, P.bc_hi, sn);
        const unsigned id = pbase + axis_off(P, jn);
        nx5[0] = __ldg(P.inf[0] + id);
        nx5[1] = __ldg(P.inf[Dir<DIR>::U] + id);
        nx5[2] = __ldg(P.inf[Dir<DIR>::V] + id);
        nx5[3] = __ldg(P.inf[Dir<DIR>::W] + id);
        nx5[4] = __ldg(P.inf[4] + id);
    }
    __device__ __forceinline__ void begin(int) {}
    __device__ __forceinline__ void hydro(int n, int& j, float& sgn, float (&v)[5]) {
        j = jn; sgn = sn;
#pragma unroll
        for (int k = 0; k < 5; ++k) v[k] = nx5[k];
        v[1] *= sgn;
        fetch(n + 1);        // overshoots by one plane at the end of the pencil: still a valid image cell
    }
    __device__ __forceinline__ void fetch_ppb(int c) {
        const int j = image_cell(c, P.n, P.bc_lo, P.bc_hi, snm);
        const unsigned id = pbase + axis_off(P, j);
#pragma unroll
        for (int k = 0; k < 10; ++k) nm[k] = __ldg(P.inf[5 + PPB_PERM[DIR][k]] + id);
    }
    __device__ __forceinline__ void ppb(int c, float (&m)[10]) {
#pragma unroll
        for (int k = 0; k < 10; ++k) m[k] = nm[k];
        m[1] *= snm; m[4] *= snm; m[6] *= snm;
        fetch_ppb(c + 1);    // one cell ahead of its use (overshoots by one at the end: still a valid image cell)
    }
    __device__ __forceinline__ void store(int i, const float (&h)[5], const float (&m)[10]) {
        const unsigned id = pbase + axis_off(P, i);
        P.outf[0][id] = h[0];
        P.outf[Dir<DIR>::U][id] = h[1];
        P.outf[Dir<DIR>::V][id] = h[2];
        P.outf[Dir<DIR>::W][id] = h[3];
        P.outf[4][id] = h[4];
#pragma unroll
        for (int k = 0; k < 10; ++k) P.outf[5 + PPB_PERM[DIR][k]][id] = m[k];
    }
    __device__ __forceinline__ void end(int) {}
    __device__ __forceinline__ void finish() {}
};

template <int DIR, int GRAV>
__global__ void __launch_bounds__(128, 3) ppm_sweep_kernel(const SweepParams P) {
    int a, b;
    if (P.brick) {      // 16 lanes = the 4x4 transverse cells of one brick; 8 bricks along a per CTA
        const int t = threadIdx.x;
        a = blockIdx.x * 32 + (t >> 4) * 4 + (t & 3);
        b = blockIdx.y * 4 + ((t >> 2) & 3);
    } else {
        a = blockIdx.x * blockDim.x + threadIdx.x;
        b = blockIdx.y;
    }
    if (a >= P.na || b >= P.nb) return;
    const unsigned wmask = __activemask();
    const int c0 = blockIdx.z * P.chunk;
    const int c1 = min(c0 + P.chunk, P.n);
    const unsigned tb = (unsigned)(a >> 2) * (unsigned)P.SBa + (unsigned)(a & 3) * (unsigned)P.SIa + (unsigned)(b >> 2) * (unsigned)P.SBb + (unsigned)(b & 3) * (unsigned)P.SIb;
    IoDirect<DIR> io(P, tb, c0 - PPM_NGHOST, c0);
    march<DIR, GRAV>(P, io, a, b, c0, c1, true, wmask);
}

// =====================================================================================================
// IoTmaX: x sweep on the brick layout.  Warp = 2 bricks adjacent in y (lane = bsel*16 + iz*4 + iy).  The TMA
// box {64 floats of a brick, 1 bx, 2 by, 1 bz, 5 fields} lands as [field][lane][4 x-cells], so every lane owns
// the 16 bytes at slot `lane` of every field: thread-private, conflict-free, whole 256-byte bricks on the wire.
// Rings: hydro fields 2 chunks (2 x 2560 B), PPB fields 2 chunks (2 x 5120 B, read three cells later),
// results 1 chunk (7680 B) written back by TMA store.  23040 B per warp.
// =====================================================================================================
constexpr int TX_ROWS = 32, TX_CH = 4;
constexpr int TX_HYD = 5 * TX_ROWS * TX_CH;           // floats per hydro chunk buffer
constexpr int TX_PPB = 10 * TX_ROWS * TX_CH;
constexpr int TX_OUT = 15 * TX_ROWS * TX_CH;
constexpr int TX_WARP_FLOATS = 2 * TX_HYD + 2 * TX_PPB + TX_OUT;   // 5760 floats = 23040 B
constexpr int TX_WARPS = 4;

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// coordinates: (element in brick = 0, bx, by, bz, field)
__device__ __forceinline__ void tma_load_brick(void* dst, const CUtensorMap* map, uint64_t* bar, int bx, int by, int bz, int f) {
    asm volatile(
        "cp.async.bulk.tensor.5d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6, %7}], [%2];"
        ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(0), "r"(bx), "r"(by), "r"(bz), "r"(f) : "memory");
}
__device__ __forceinline__ void tma_store_brick(const CUtensorMap* map, const void* src, int bx, int by, int bz, int f) {
    asm volatile("cp.async.bulk.tensor.5d.global.shared::cta.tile.bulk_group [%0, {%2, %3, %4, %5, %6}], [%1];"
                 ::"l"(map), "r"(smem_u32(src)), "r"(0), "r"(bx), "r"(by), "r"(bz), "r"(f) : "memory");
}
__device__ __forceinline__ void tma_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void tma_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void tma_wait_all0() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

struct IoTmaX {
    const SweepParams& P;
    const CUtensorMap* tin;
    const CUtensorMap* tout;
    float* hyd;          // warp's hydro ring [2][5][32][4]
    float* ppbuf;        // warp's PPB ring   [2][10][32][4]
    float* outb;         // warp's result chunk [15][32][4]
    uint64_t* bar;       // [0..1] hydro ring, [2..3] PPB ring
    const int lane, by0, bz;
    const int k0, kend;  // first / last chunk index (chunk k = brick bx = k = cells 4k .. 4k+3)
    bool store_pending;

    __device__ __forceinline__ IoTmaX(const SweepParams& P_, const CUtensorMap* ti, const CUtensorMap* to, float* wsm, uint64_t* wbar,
                                      int lane_, int by0_, int bz_, int c0, int c1)
        : P(P_), tin(ti), tout(to), hyd(wsm), ppbuf(wsm + 2 * TX_HYD), outb(wsm + 2 * TX_HYD + 2 * TX_PPB), bar(wbar),
          lane(lane_), by0(by0_), bz(bz_), k0(c0 / TX_CH - 1), kend(c1 / TX_CH), store_pending(false) {
        if (lane == 0) {
            issue_hydro(k0); issue_ppb(k0);
            if (k0 + 1 <= kend) { issue_hydro(k0 + 1); issue_ppb(k0 + 1); }
        }
    }
    // brick index bx holding chunk k (ghost chunks map onto their periodic / mirror image; mirrored ones are read reversed)
    __device__ __forceinline__ int chunk_bx(int k, bool& rev) const {
        rev = false;
        const int nk = P.nbrick_d;
        if (k < 0) { if (P.bc_lo == PPM_BC_PERIODIC) return nk - 1; rev = true; return 0; }
        if (k >= nk) { if (P.bc_hi == PPM_BC_PERIODIC) return 0; rev = true; return nk - 1; }
        return k;
    }
    __device__ __forceinline__ void issue_hydro(int k) {
        bool rev; const int bx = chunk_bx(k, rev);
        const int bsel = (k - k0) & 1;
        mbar_expect_tx(bar + bsel, TX_HYD * 4);
        tma_load_brick(hyd + bsel * TX_HYD, tin, bar + bsel, bx, by0, bz, 0);
    }
    __device__ __forceinline__ void issue_ppb(int k) {
        bool rev; const int bx = chunk_bx(k, rev);
        const int bsel = (k - k0) & 1;
        mbar_expect_tx(bar + 2 + bsel, TX_PPB * 4);
        tma_load_brick(ppbuf + bsel * TX_PPB, tin, bar + 2 + bsel, bx, by0, bz, 5);
        tma_load_brick(ppbuf + bsel * TX_PPB + TX_HYD, tin, bar + 2 + bsel, bx, by0, bz, 10);
    }
    __device__ __forceinline__ void begin(int n) {
        if ((n & 3) == 0) {                                   // first cell of hydro chunk k
            const int k = n >> 2;
            mbar_wait(bar + ((k - k0) & 1), ((k - k0) >> 1) & 1);
        }
        const int c = n - 3;                                   // PPB cell of this iteration
        if ((c & 3) == 0 || c == 4 * k0 + 3) {                 // first PPB cell read from its chunk
            const int k = c >> 2;
            if (k >= k0) mbar_wait(bar + 2 + ((k - k0) & 1), ((k - k0) >> 1) & 1);
        }
    }
    __device__ __forceinline__ void hydro(int n, int& j, float& sgn, float (&v)[5]) {
        const int k = n >> 2;
        bool rev; const int bx = chunk_bx(k, rev);
        int s = n & 3;
        if (rev) s = 3 - s;
        sgn = rev ? -1.0f : 1.0f;
        j = bx * TX_CH + s;
        const float* src = hyd + ((k - k0) & 1) * TX_HYD + lane * TX_CH + s;
        v[0] = src[0];
        v[1] = sgn * src[1 * TX_ROWS * TX_CH];                 // normal velocity ux is field 1 (odd under mirror)
        v[2] = src[2 * TX_ROWS * TX_CH];
        v[3] = src[3 * TX_ROWS * TX_CH];
        v[4] = src[4 * TX_ROWS * TX_CH];
    }
    __device__ __forceinline__ void ppb(int c, float (&m)[10]) {
        const int k = c >> 2;
        bool rev; chunk_bx(k, rev);
        int s = c & 3;
        if (rev) s = 3 - s;
        const float sgn = rev ? -1.0f : 1.0f;
        const float* src = ppbuf + ((k - k0) & 1) * TX_PPB + lane * TX_CH + s;
#pragma unroll
        for (int q = 0; q < 10; ++q) m[q] = src[PPB_PERM[0][q] * TX_ROWS * TX_CH];
        m[1] *= sgn; m[4] *= sgn; m[6] *= sgn;
    }
    __device__ __forceinline__ void store(int i, const float (&h)[5], const float (&m)[10]) {
        const int s = i & 3;
        if (s == 0 && store_pending) {                         // the previous chunk's TMA store must have read outb
            if (lane == 0) tma_wait_read0();
            __syncwarp();
            store_pending = false;
        }
        float* dst = outb + lane * TX_CH + s;
#pragma unroll
        for (int f = 0; f < 5; ++f) dst[f * TX_ROWS * TX_CH] = h[f];
#pragma unroll
        for (int q = 0; q < 10; ++q) dst[(5 + PPB_PERM[0][q]) * TX_ROWS * TX_CH] = m[q];
        if (s == 3) {
            fence_async_smem();                                // generic-proxy writes -> visible to the async proxy
            __syncwarp();
            if (lane == 0) {
                const int bx = i >> 2;
                tma_store_brick(tout, outb, bx, by0, bz, 0);
                tma_store_brick(tout, outb + TX_HYD, bx, by0, bz, 5);
                tma_store_brick(tout, outb + 2 * TX_HYD, bx, by0, bz, 10);
                tma_commit();
            }
            store_pending = true;
        }
    }
    __device__ __forceinline__ void end(int n) {
        // ring refills: a buffer is free once every lane has taken its last value from it
        if ((n & 3) == 3) {                                    // hydro chunk k = n>>2 fully consumed
            const int k = n >> 2;
            __syncwarp();
            if (lane == 0 && k + 2 <= kend) issue_hydro(k + 2);
        }
        const int c = n - 3;
        if ((c & 3) == 3) {                                    // PPB chunk k = c>>2 fully consumed
            const int k = c >> 2;
            __syncwarp();
            if (lane == 0 && k >= k0 && k + 2 <= kend) issue_ppb(k + 2);
        }
    }
    __device__ __forceinline__ void finish() {
        if (lane == 0) tma_wait_all0();                        // smem must outlive the last bulk store
        __syncwarp();
    }
};

template <int GRAV>
__global__ void __launch_bounds__(TX_WARPS * 32, 2) ppm_sweep_x_tma_kernel(const SweepParams P, const __grid_constant__ CUtensorMap tin,
                                                                        const __grid_constant__ CUtensorMap tout) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float* sm = reinterpret_cast<float*>(smem_raw);
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem_raw + (size_t)TX_WARPS * TX_WARP_FLOATS * 4);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x < TX_WARPS * 4) mbar_init(bars + threadIdx.x, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    fence_async_smem();
    __syncthreads();
    const int by0 = (blockIdx.x * TX_WARPS + warp) * 2;        // the warp's two bricks: by0, by0+1 at bz
    if (by0 * 4 >= P.na) return;                               // whole warp out of range (no block-wide sync below)
    const int bz = blockIdx.y;
    const int a = (by0 + (lane >> 4)) * 4 + (lane & 3);        // y
    const int b = bz * 4 + ((lane >> 2) & 3);                  // z
    const int c0 = blockIdx.z * P.chunk;
    const int c1 = min(c0 + P.chunk, P.n);
    IoTmaX io(P, &tin, &tout, sm + warp * TX_WARP_FLOATS, bars + warp * 4, lane, by0, bz, c0, c1);
    march<0, GRAV>(P, io, a, b, c0, c1, a < P.na, 0xffffffffu);
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

constexpr size_t TX_SMEM = (size_t)TX_WARPS * TX_WARP_FLOATS * 4 + TX_WARPS * 4 * sizeof(uint64_t);

template <int GRAV>
cudaError_t launch_x_tma(const SweepParams& P, const CUtensorMap& tin, const CUtensorMap& tout, dim3 grid, cudaStream_t st) {
    static bool attr_done = false;
    if (!attr_done) {
        cudaError_t e = cudaFuncSetAttribute(ppm_sweep_x_tma_kernel<GRAV>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TX_SMEM);
        if (e != cudaSuccess) return e;
        attr_done = true;
    }
    ppm_sweep_x_tma_kernel<GRAV><<<grid, TX_WARPS * 32, TX_SMEM, st>>>(P, tin, tout);
    return cudaGetLastError();
}

}  // namespace

// ---- host: tensor maps for the x-sweep TMA path -------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

bool ppm_make_xmaps(ppm_ctx* c) {
    c->tma_ok = 0;
    const ppm_params& p = c->prm;
    if (c->layout != 1) return false;                           // the TMA path stages bricks
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn ||
        qres != cudaDriverEntryPointSuccess) {
        cudaGetLastError();
        return false;
    }
    EncodeTiledFn enc = (EncodeTiledFn)fn;
    const cuuint64_t nbx = p.nx / 4, nby = p.ny / 4, nbz = p.nz / 4;
    const cuuint64_t dims[5] = {64, nbx, nby, nbz, PPM_NFIELDS};
    const cuuint64_t strides[4] = {256, 256 * nbx, 256 * nbx * nby, 256 * nbx * nby * nbz};
    const cuuint32_t box[5] = {64, 1, 2, 1, 5};
    const cuuint32_t estr[5] = {1, 1, 1, 1, 1};
    for (int b = 0; b < 2; ++b) {
        CUresult r = enc(reinterpret_cast<CUtensorMap*>(c->xmap[b]), CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 5, c->buf[b], dims, strides, box, estr,
                         CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                         CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return false;
    }
    c->tma_ok = 1;
    return true;
}

cudaError_t ppm_launch_sweep(ppm_ctx* c, int axis, double dt) {
    const ppm_params& p = c->prm;
    const long long nx = p.nx, ny = p.ny, nz = p.nz;
    SweepParams P;
    const float* in = c->buf[c->cur];
    float* out = c->buf[c->cur ^ 1];
    P.ncell = nx * ny * nz;
    for (int f = 0; f < PPM_NFIELDS; ++f) { P.inf[f] = in + f * P.ncell; P.outf[f] = out + f * P.ncell; }
    const int ext[3] = {p.nx, p.ny, p.nz};
    const int ia = (axis == 0) ? 1 : 0;       // thread-mapped transverse axis
    const int ib = (axis == 2) ? 1 : 2;       // second transverse axis
    P.n = ext[axis]; P.na = ext[ia]; P.nb = ext[ib];
    long long SB[3]; int SI[3];
    if (c->layout == 1) {
        const long long nbx = nx / 4, nby = ny / 4;
        SB[0] = 64; SB[1] = 64 * nbx; SB[2] = 64 * nbx * nby;
        SI[0] = 1; SI[1] = 4; SI[2] = 16;
    } else {
        const long long str[3] = {1, nx, nx * ny};
        for (int d = 0; d < 3; ++d) { SB[d] = 4 * str[d]; SI[d] = (int)str[d]; }
    }
    P.SBd = SB[axis]; P.SBa = SB[ia]; P.SBb = SB[ib];
    P.SId = SI[axis]; P.SIa = SI[ia]; P.SIb = SI[ib];
    P.brick = c->layout;
    P.nbrick_d = P.n / 4;
    P.bc_lo = p.bc[2 * axis]; P.bc_hi = p.bc[2 * axis + 1];
    const bool use_tma = (axis == 0) && c->tma_ok && !c->force_direct;
    int chunk = c->chunk > 0 ? c->chunk : P.n;
    if (use_tma) chunk = (chunk + 3) / 4 * 4;
    if (chunk > P.n) chunk = P.n;
    P.chunk = chunk;
    P.dt = (float)dt; P.dx = (float)p.dx; P.dtdx = (float)(dt / p.dx); P.inv_dx = (float)(1.0 / p.dx);
    P.gamma = (float)p.gamma; P.rho_floor = (float)p.rho_floor; P.p_floor = (float)p.p_floor;
    P.tab_n = p.grav.n; P.s0 = (float)p.grav.s0; P.inv_ds = (float)(p.grav.kind != PPM_GRAV_NONE ? 1.0 / p.grav.ds : 0.0);
    P.cen_d = (float)p.grav.center[axis]; P.cen_a = (float)p.grav.center[ia]; P.cen_b = (float)p.grav.center[ib];
    P.tab = c->tab;
    P.flag = c->flag;
    const int nchunks = (P.n + chunk - 1) / chunk;
    cudaError_t e;
    if (use_tma) {
        const CUtensorMap& tin = *reinterpret_cast<const CUtensorMap*>(c->xmap[c->cur]);
        const CUtensorMap& tout = *reinterpret_cast<const CUtensorMap*>(c->xmap[c->cur ^ 1]);
        dim3 grid((P.na + TX_WARPS * 8 - 1) / (TX_WARPS * 8), P.nb / 4, nchunks);   // CTA = 8 bricks along y, 1 along z
        if (p.grav.kind == PPM_GRAV_NONE) e = launch_x_tma<PPM_GRAV_NONE>(P, tin, tout, grid, c->stream);
        else if (p.grav.kind == PPM_GRAV_CONST_Z) e = launch_x_tma<PPM_GRAV_CONST_Z>(P, tin, tout, grid, c->stream);
        else e = launch_x_tma<PPM_GRAV_RADIAL>(P, tin, tout, grid, c->stream);
    } else {
        dim3 block(128, 1, 1);
        dim3 grid = c->layout == 1 ? dim3((P.na + 31) / 32, (P.nb + 3) / 4, nchunks) : dim3((P.na + 127) / 128, P.nb, nchunks);
        if (axis == 0) e = launch_dir<0>(P, p.grav.kind, grid, block, c->stream);
        else if (axis == 1) e = launch_dir<1>(P, p.grav.kind, grid, block, c->stream);
        else e = launch_dir<2>(P, p.grav.kind, grid, block, c->stream);
    }
    if (e == cudaSuccess) { c->cur ^= 1; c->launches += 1; }
    return e;
}
