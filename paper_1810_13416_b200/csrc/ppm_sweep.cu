// ppm_sweep.cu — the fused PPM hydro + PPB remap sweep kernels (sm_100a).
//
// One thread owns one grid pencil (pencils are independent within a 1-D pass) and
// marches along the sweep axis with a short sliding window held on chip — the paper's pipelined pencil
// update with a barrel shift (Fig. 7), re-designed for brick records with SoA fields: lanes run along
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
// State layout in HBM: brick records — the grid is cut into bricks of 4x4x4 cells and a brick holds all 15
// fields of its 64 cells, field-major: [bz][by][bx][15][4z][4y][4x], 3840 B per brick (ppm_internal.h).  The
// paper's briquettes answer the same problem; here the fields stay separate inside the record
// (SoA), so a warp's 32 pencils = 2 brick columns x (4x4 transverse cells) and no on-chip transposition or
// 16||16 splice (L118, L124) is ever needed.
//
// Two data paths feed the same marching body:
//   IoBulk    (default; extent along the sweep axis a multiple of 4) every direction: the hydro part (1280 B) and
//             the PPB part (2560 B) of a brick are 1-D bulk copies (cp.async.bulk + mbarrier) into per-warp rings
//             in shared memory; results are written in place over the brick's own input and shipped back with a
//             bulk store.  DRAM only ever sees whole 1280/2560-byte runs; no load waits in a register.
//   IoDirect  (any extent) straight global loads / stores, 16 lanes per 64-byte brick layer, next plane
//             software-prefetched into registers.
//
// fp32 arithmetic.  rho and p are carried as perturbations to the base state; every
// difference of nearly equal numbers is taken between perturbation-sized quantities only ("explicitly
// cancel out all large contributions", L35): the Newton iteration runs on p*' = p* - p0f, the update
// adds increments to rho', p' instead of rebuilding them from E.
#include <stdlib.h>
#include <string.h>

#include <type_traits>

#include "ppm_internal.h"

#ifndef PPM_MARCH_UNROLL
#define PPM_MARCH_UNROLL 1
#endif
// bulk path: cells of the steady-state marching loop per loop body (1, 2 or 4 = one brick with compile-time phases)
#ifndef PPM_FAST_UNROLL
#define PPM_FAST_UNROLL 1
#endif
// warp-uniform shortcuts past work whose outcome is known for every lane (no shock near, star state at the face,
// Newton converged, PPB polynomial inside its bounds); a bit mask, 0 = always the general code (A/B knob)
#ifndef PPM_NEWTON_NESTED
#define PPM_NEWTON_NESTED 1     // Newton iterations 2..5 as nested ifs instead of a loop (round 2: -1.6 %, profiles/r2_experiments.md)
#endif
#ifndef PPM_UNIFORM_FAST
#define PPM_UNIFORM_FAST 3      // bits: 1 flattening, 2 converged W_K, 4 star state, 8 PPB theta  (3: -0.8 % against 2 on the final code)
#endif
// direct-path CTA shape (build knobs): threads per CTA (a multiple of 16 = one brick column; the kernel uses no
// shared memory and no block-wide sync, so the CTA size only sets the granularity of occupancy) and the register
// cap per thread (65536 / (cap rounded up to 8) / 32 = resident warps per SM)
#ifndef PPM_CTA
#define PPM_CTA 128
#endif
#ifndef PPM_MAXREG
#define PPM_MAXREG 168
#endif
// direct path: whole brick records this many bricks ahead along the pencil are pulled into L2 with one bulk
// prefetch per half warp (0 = off)
// bulk path: warps per CTA (1, 2, 3, 4, 6 or 12: 12 warps stay resident per SM)
#ifndef PPM_BULK_WARPS
#define PPM_BULK_WARPS 4
#endif
#ifndef PPM_K10_PARAM
#define PPM_K10_PARAM 1
#endif
// steady-state body: bulk copies issued by the whole warp under a leader predicate instead of inside `if (lane == 0)` (A/B knob)
#ifndef PPM_PRED_COPIES
#define PPM_PRED_COPIES 1
#endif
#ifndef PPM_PPB_PAIRS
#define PPM_PPB_PAIRS 0      // 1: shift the (a0,a1), (a2,f0) pairs with packed FMA-pipe copies too (measured slower: 12.87 vs 12.83 ms)
#endif
// warp-uniform shortcut past the PPB remap where FV is uniform (same values; A/B knob)
#ifndef PPM_FV_SKIP
#define PPM_FV_SKIP 1
#endif
#ifndef PPM_PREFETCH_BRICKS
#define PPM_PREFETCH_BRICKS 1
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
// streaming read that leaves the (small: L1 is carved out as shared memory) L1 to the gravity-table lines
__device__ __forceinline__ float ld_noalloc(const float* p) { float v; asm volatile("ld.global.nc.L1::no_allocate.f32 %0, [%1];" : "=f"(v) : "l"(p)); return v; }
// the detector field F~ (3-D flattening mode): a brick's 256 bytes are read in four iterations, 64 bytes (z sweep: one row) or 16
// scattered 4-byte pieces of every sector (x, y sweeps) at a time — with L1 allocation the sectors are fetched once per brick
#ifndef PPM_FLAT_L1
#define PPM_FLAT_L1 1
#endif
__device__ __forceinline__ float ld_flat(const float* p) { return PPM_FLAT_L1 ? __ldg(p) : ld_noalloc(p); }
__device__ __forceinline__ float med3(float a, float b, float c) { return fmaxf(fminf(a, b), fminf(fmaxf(a, b), c)); }
__device__ __forceinline__ float rcp(float x) { return __fdividef(1.0f, x); }
__device__ __forceinline__ float fdiv(float a, float b) { return __fdividef(a, b); }
__device__ __forceinline__ float fsqrt(float x) { return x * rsqrtf(fmaxf(x, 1e-37f)); }

// ---- packed fp32 pairs (sm_100a FADD2 / FMUL2 / FFMA2) --------------------------------------------------
// The sweep is bound by instruction issue, not by the FP32 lanes: one f32x2 instruction does the work of two
// scalar ones in one issue slot.  A v2 lives in an aligned register pair; ptxas folds negation, |x|, the
// (-,+) / (+,-) sign patterns, half swaps and scalar broadcasts into operand modifiers, and min/max/select on
// a half are ordinary scalar instructions on that register — so packing costs no extra moves.
struct v2 { float x, y; };
__device__ __forceinline__ unsigned long long pk(v2 a) { unsigned long long r; asm("mov.b64 %0, {%1,%2};" : "=l"(r) : "f"(a.x), "f"(a.y)); return r; }
__device__ __forceinline__ v2 up(unsigned long long a) { v2 r; asm("mov.b64 {%0,%1}, %2;" : "=f"(r.x), "=f"(r.y) : "l"(a)); return r; }
__device__ __forceinline__ v2 operator+(v2 a, v2 b) { unsigned long long r; asm("add.rn.ftz.f32x2 %0, %1, %2;" : "=l"(r) : "l"(pk(a)), "l"(pk(b))); return up(r); }
__device__ __forceinline__ v2 operator-(v2 a, v2 b) { unsigned long long r; asm("sub.rn.ftz.f32x2 %0, %1, %2;" : "=l"(r) : "l"(pk(a)), "l"(pk(b))); return up(r); }
__device__ __forceinline__ v2 operator*(v2 a, v2 b) { unsigned long long r; asm("mul.rn.ftz.f32x2 %0, %1, %2;" : "=l"(r) : "l"(pk(a)), "l"(pk(b))); return up(r); }
__device__ __forceinline__ v2 fma2(v2 a, v2 b, v2 c) { unsigned long long r; asm("fma.rn.ftz.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(pk(a)), "l"(pk(b)), "l"(pk(c))); return up(r); }
__device__ __forceinline__ v2 mk(float x, float y) { v2 r; r.x = x; r.y = y; return r; }
__device__ __forceinline__ v2 bc(float s) { return mk(s, s); }                 // broadcast
__device__ __forceinline__ v2 operator*(v2 a, float s) { return a * bc(s); }
__device__ __forceinline__ v2 operator-(v2 a) { return mk(-a.x, -a.y); }
__device__ __forceinline__ v2 np(v2 a) { return mk(-a.x, a.y); }              // (-,+) sign pattern
__device__ __forceinline__ v2 swp(v2 a) { return mk(a.y, a.x); }
__device__ __forceinline__ v2 abs2(v2 a) { return mk(fabsf(a.x), fabsf(a.y)); }
__device__ __forceinline__ float hsum(v2 a) { return a.x + a.y; }
// A register-pair copy as ONE instruction on the FMA pipe (x * 1 under flush-to-zero).  The sliding windows of the
// marching loop are shifted once per cell; as plain copies they are ~130 MOVs on the half-rate ALU pipe, issued in one
// burst that starves the other warps' min/max/select work.
#ifndef PPM_PACKED_MOVES
#define PPM_PACKED_MOVES 1
#endif
#ifndef PPM_PM
#define PPM_PM 5
#endif
#define MV5B(x) ((PPM_PM & 1) ? mv5(x) : (x))
#define MV5C(x) ((PPM_PM & 2) ? mv5(x) : (x))
#define MV2D(x) ((PPM_PM & 4) ? mv2(x) : (x))
__device__ __forceinline__ v2 mv2(v2 a) {
#if PPM_PACKED_MOVES
    unsigned long long r; asm("mul.rn.ftz.f32x2 %0, %1, %2;" : "=l"(r) : "l"(pk(a)), "l"(pk(mk(1.0f, 1.0f)))); return up(r);
#else
    return a;
#endif
}

// the five interpolated variables of a cell: A = (rho', p'), B = (v, w) transverse, u normal
struct V5 { v2 A, B; float u; };
__device__ __forceinline__ V5 operator+(const V5& a, const V5& b) { V5 r; r.A = a.A + b.A; r.B = a.B + b.B; r.u = a.u + b.u; return r; }
__device__ __forceinline__ V5 operator-(const V5& a, const V5& b) { V5 r; r.A = a.A - b.A; r.B = a.B - b.B; r.u = a.u - b.u; return r; }
__device__ __forceinline__ V5 operator*(const V5& a, const V5& b) { V5 r; r.A = a.A * b.A; r.B = a.B * b.B; r.u = a.u * b.u; return r; }
__device__ __forceinline__ V5 operator*(const V5& a, float s) { V5 r; r.A = a.A * bc(s); r.B = a.B * bc(s); r.u = a.u * s; return r; }
__device__ __forceinline__ V5 fma5(const V5& a, const V5& b, const V5& c) { V5 r; r.A = fma2(a.A, b.A, c.A); r.B = fma2(a.B, b.B, c.B); r.u = fmaf(a.u, b.u, c.u); return r; }
__device__ __forceinline__ V5 fma5(const V5& a, float s, const V5& c) { V5 r; r.A = fma2(a.A, bc(s), c.A); r.B = fma2(a.B, bc(s), c.B); r.u = fmaf(a.u, s, c.u); return r; }
__device__ __forceinline__ V5 abs5(const V5& a) { V5 r; r.A = abs2(a.A); r.B = abs2(a.B); r.u = fabsf(a.u); return r; }
__device__ __forceinline__ V5 bc5(float s) { V5 r; r.A = bc(s); r.B = bc(s); r.u = s; return r; }
__device__ __forceinline__ V5 zero5() { V5 r; r.A = bc(0.f); r.B = bc(0.f); r.u = 0.f; return r; }
// window shift of a cell's five variables: the two pairs as packed copies
__device__ __forceinline__ V5 mv5(const V5& a) { V5 r; r.A = mv2(a.A); r.B = mv2(a.B); r.u = a.u; return r; }
template <class F> __device__ __forceinline__ V5 map3(const V5& a, const V5& b, const V5& c, F f) {
    V5 r; r.A = mk(f(a.A.x, b.A.x, c.A.x), f(a.A.y, b.A.y, c.A.y)); r.B = mk(f(a.B.x, b.B.x, c.B.x), f(a.B.y, b.B.y, c.B.y)); r.u = f(a.u, b.u, c.u); return r;
}

// image of a cell / face index outside [0, n) under the boundary condition (C3).  The index is the same for
// every lane of a warp; all but the 8 ghost iterations of a pencil take the first return.
__device__ __forceinline__ int image_cell(int i, int n, int bc_lo, int bc_hi, float& sgn) {
    sgn = 1.0f;
    if ((unsigned)i < (unsigned)n) return i;
    const int bcx = (i < 0) ? bc_lo : bc_hi;
    if (bcx == PPM_BC_PERIODIC) {
        i += (i < 0) ? n : -n;
        if ((unsigned)i >= (unsigned)n) i = ((i % n) + n) % n;      // fewer cells than ghosts
        return i;
    }
    sgn = -1.0f;
    const int s = (i < 0) ? (-1 - i) : (2 * n - 1 - i);
    return min(max(s, 0), n - 1);
}
__device__ __forceinline__ int image_face(int f, int n, int bc_lo, int bc_hi) {
    if ((unsigned)f < (unsigned)n) return f;
    if (f == n) return (bc_hi == PPM_BC_PERIODIC) ? 0 : f;
    const int bcx = (f < 0) ? bc_lo : bc_hi;
    if (bcx == PPM_BC_HALO) return f;                                 // a neighbour's cells: the face is where it is
    if (bcx == PPM_BC_PERIODIC) {
        f += (f < 0) ? n : -n;
        if ((unsigned)f >= (unsigned)n) f = ((f % n) + n) % n;
        return f;
    }
    const int s = (f < 0) ? -f : 2 * n - f;
    return min(max(s, 0), n);
}

// ---- base state (C1) -----------------------------------------------------------------------------
// table node k: {rho0, p0, g, 0} — (rho0, p0) is an aligned pair
struct Base { v2 rp; float g; };

// interval index and weight of table position s
__device__ __forceinline__ int table_interval(const SweepParams& P, float s, float& w) {
    const float t = (s - P.s0) * P.inv_ds;
    int k = (int)floorf(t);
    k = min(max(k, 0), P.tab_n - 2);
    w = t - (float)k;
    return k;
}
// one load per quantity: the interval records hold the node value and the difference to the next node
__device__ __forceinline__ v2 table_rp(const SweepParams& P, float s) {
    float w;
    const int k = table_interval(P, s, w);
    const float4 a = __ldg(P.tabp + k);
    return fma2(bc(w), mk(a.z, a.w), mk(a.x, a.y));
}
__device__ __forceinline__ Base table_at(const SweepParams& P, float s) {
    float w;
    const int k = table_interval(P, s, w);
    const float4 a = __ldg(P.tabp + k);
    const float2 g = __ldg(P.tabg + k);
    Base o;
    o.rp = fma2(bc(w), mk(a.z, a.w), mk(a.x, a.y));
    o.g = fmaf(w, g.y, g.x);
    return o;
}

// per-thread geometry for the base state
template <int DIR, int GRAV> struct Geo {
    float t2;      // RADIAL: squared transverse distance from the centre
    Base cst;      // CONST_Z, DIR != 2: the base state is constant along the pencil
    __device__ __forceinline__ void init(const SweepParams& P, int a, int b) {
        t2 = 0.f; cst.rp = bc(0.f); cst.g = 0.f;
        if (GRAV == PPM_GRAV_RADIAL) {
            // (org: global index of the grid's cell 0 — a sub-domain of a brick decomposition evaluates the base state at the
            //  same global positions, with the same arithmetic, as the undivided grid; 0 otherwise)
            float xa = ((float)(a + P.org_a) + 0.5f) * P.dx - P.cen_a, xb = ((float)(b + P.org_b) + 0.5f) * P.dx - P.cen_b;
            t2 = xa * xa + xb * xb;
        } else if (GRAV == PPM_GRAV_CONST_Z && DIR != 2) {
            float4 v = __ldg(P.tab + 2 * b + 2 * PPM_NGHOST + 1);   // b is the z index for x- and y-sweeps
            cst.rp = mk(v.x, v.y); cst.g = 0.f;                     // no acceleration along x or y
        }
    }
    // cell centre with image index j (sign sgn for the odd normal acceleration)
    __device__ __forceinline__ Base cell(const SweepParams& P, int j, float sgn) const {
        Base o; o.rp = bc(0.f); o.g = 0.f;
        if (GRAV == PPM_GRAV_CONST_Z) {
            if (DIR == 2) { float4 v = __ldg(P.tab + 2 * j + 2 * PPM_NGHOST + 1); o.g = sgn * v.z; o.rp = mk(v.x, v.y); }
            else o = cst;
        } else if (GRAV == PPM_GRAV_RADIAL) {
            float xd = ((float)(j + P.org_d) + 0.5f) * P.dx - P.cen_d;
            float r2 = fmaf(xd, xd, t2);
            float ir = rsqrtf(fmaxf(r2, 1e-30f));
            o = table_at(P, r2 * ir);
            o.g = sgn * o.g * xd * ir;
        }
        return o;
    }
    // face with image index f (position f*dx along the sweep axis): (rho0, p0)
    __device__ __forceinline__ v2 face(const SweepParams& P, int f) const {
        v2 o = bc(0.f);
        if (GRAV == PPM_GRAV_CONST_Z) {
            if (DIR == 2) { float4 v = __ldg(P.tab + 2 * f + 2 * PPM_NGHOST); o = mk(v.x, v.y); }
            else o = cst.rp;
        } else if (GRAV == PPM_GRAV_RADIAL) {
            float xd = (float)(f + P.org_d) * P.dx - P.cen_d;
            float r2 = fmaf(xd, xd, t2);
            o = table_rp(P, fsqrt(r2));
        }
        return o;
    }
};

// ---- H2 + H3: limited parabola blended with the unlimited one ------------------------------------
// Lc, Rc: face values already clamped between the neighbouring cell means (per-face medians); fl, fr the
// unlimited faces; om the smoothness weight.  With a = Rc - q0, b = q0 - Lc (same sign unless the cell is an
// extremum): Delta = a + b, q6 = 3(b - a), so the Colella-Woodward overshoot tests Delta*q6 > Delta^2 and
// Delta*q6 < -Delta^2 are |b| > 2|a| and |a| > 2|b|, and the corrected faces are q0 - 2a and q0 + 2b.
__device__ __forceinline__ void parabola(const V5& q0, const V5& Lc, const V5& Rc, const V5& fl, const V5& fr, const V5& om, V5& L, V5& R) {
    const V5 a = Rc - q0, b = q0 - Lc;
    const V5 pr = a * b;
    const V5 a2 = a + a, b2 = b + b;
    const V5 La = q0 - a2, Ra = q0 + b2;
    // L2: extremum -> q0; |b| > |2a| -> q0 - 2a; else Lc.   (selects are per element)
    V5 L2, R2;
#define PPM_SEL(E) \
    { const bool ext = pr.E <= 0.0f; \
      const float l = (fabsf(b.E) > fabsf(a2.E)) ? La.E : Lc.E; \
      const float r = (fabsf(a.E) > fabsf(b2.E)) ? Ra.E : Rc.E; \
      L2.E = ext ? q0.E : l; R2.E = ext ? q0.E : r; }
    PPM_SEL(A.x) PPM_SEL(A.y) PPM_SEL(B.x) PPM_SEL(B.y) PPM_SEL(u)
#undef PPM_SEL
    L = fma5(om, L2 - fl, fl);
    R = fma5(om, R2 - fr, fr);
}

// ---- P4: exact projection of up to three pieces onto the Legendre basis ---------------------------
// pre-limited coefficients of one cell in local family order, stored as the pairs the remap uses
struct PpbCell { v2 a01, a2f; v2 bc0, bc1, de; };   // a01 = (a0, a1), a2f = (a2, f0), bc0 = (b0, c0), bc1 = (b1, c1), de = (d0, e0): all pairs, shifted as such
__device__ __forceinline__ void mv_ppb(PpbCell& d, const PpbCell& s) { d.a01 = PPM_PPB_PAIRS ? mv2(s.a01) : s.a01; d.a2f = PPM_PPB_PAIRS ? mv2(s.a2f) : s.a2f; d.bc0 = mv2(s.bc0); d.bc1 = mv2(s.bc1); d.de = mv2(s.de); }

// S[0..2]: cells i-1, i, i+1 (masses per dx rm, r0, rp); dl, dr = mass per dx through the left / right
// face (positive rightward).  The two donor pieces (from i-1 and from i+1) run as one packed computation for
// the degree-2 family; the (b,c) and (d,e) families are packed inside every piece.
// irm, ir0, irp: reciprocals of the three masses; rn, irn: the cell's new mass per dx (= r0 - dr + dl; the caller has it
// as the updated density) and its reciprocal.
// CHECK: the new mass may vanish (PPB-only sweeps: rn = 1 - dt du/dx), the cell then keeps its coefficients; the full step needs
// no test: its new density is never below rho_floor, which ppm_create keeps above PPM_TINY.
template <bool CHECK>
__device__ __forceinline__ void ppb_remap(const PpbCell (&S)[3], float irm, float ir0, float irp, float rn, float irn, float dl, float dr, float (&out)[10]) {
    const bool ok = !CHECK || rn > PPM_TINY;
    const float dln = fmaxf(-dl, 0.f), drp = fmaxf(dr, 0.f);
    const v2 dD = mk(fmaxf(dl, 0.f), fmaxf(-dr, 0.f));      // donated mass: from the left cell, from the right cell
    const v2 irD = mk(irm, irp);
    // piece geometry: new-coordinate midpoint x, half width h; old-coordinate midpoint s, slope beta
    const v2 hD = dD * bc(0.5f * irn);                       // half widths of the donor pieces in the new cell
    const v2 xD = fma2(hD, mk(1.f, -1.f), mk(-0.5f, 0.5f));
    const v2 sD = fma2(dD * irD, mk(-0.5f, 0.5f), mk(0.5f, -0.5f));
    const v2 bD = irD * bc(rn);
    const float h1 = 0.5f - hD.x - hD.y, x1 = hD.x - hD.y, s1 = 0.5f * (dln - drp) * ir0, b1 = rn * ir0;
    // powers of the half width: w = 2h, w2 = 2h^3/3, w4 = 2h^5/5
    const v2 h2D = hD * hD, wD = hD + hD, w2D = (wD * h2D) * bc(1.0f / 3.0f), w4D = (w2D * h2D) * bc(0.6f);
    const float h21 = h1 * h1, w1 = h1 + h1, w21 = w1 * h21 * (1.0f / 3.0f), w41 = w21 * h21 * 0.6f;
    const v2 x2D = fma2(xD, xD, bc(-1.0f / 12.0f)), s2D = fma2(sD, sD, bc(-1.0f / 12.0f));
    const float x21 = fmaf(x1, x1, -1.0f / 12.0f), s21 = fmaf(s1, s1, -1.0f / 12.0f);
    // reference constants (own cell's degree-0 coefficients): projecting a constant is exact, so only
    // deviations from it are integrated (keeps fp32 round-off at the size of the variation)
    const float refA = S[1].a01.x;
    const v2 refBC = S[1].bc0;
    // ---- degree-2 family: donors packed (x = from i-1, y = from i+1), own piece scalar
    float a0, a1, a2;
    {
        const v2 c0 = mk(S[0].a01.x, S[2].a01.x), c1 = mk(S[0].a01.y, S[2].a01.y), c2 = mk(S[0].a2f.x, S[2].a2f.x);
        const v2 E2 = (c2 * bD) * bD, E1 = bD * fma2(c2 + c2, sD, c1);
        const v2 E0 = (c0 - bc(refA)) + fma2(c1, sD, c2 * s2D);
        const v2 J0 = fma2(w2D, E2, wD * E0), J1 = w2D * E1, J2 = fma2(w4D, E2, w2D * E0);
        const v2 A1 = fma2(xD, J0, J1), A2 = fma2(x2D, J0, fma2(xD + xD, J1, J2));
        const float d1 = S[1].a01.y, d2 = S[1].a2f.x;
        const float e2 = d2 * b1 * b1, e1 = b1 * fmaf(2.0f * d2, s1, d1);
        const float e0 = fmaf(d1, s1, d2 * s21);
        const float j0 = fmaf(w21, e2, w1 * e0), j1 = w21 * e1, j2 = fmaf(w41, e2, w21 * e0);
        a0 = hsum(J0) + j0;
        a1 = hsum(A1) + fmaf(x1, j0, j1);
        a2 = hsum(A2) + fmaf(x21, j0, fmaf(2.0f * x1, j1, j2));
    }
    // ---- the two degree-1 families (b, c) and the degree-0 pair (d, e), packed per piece; f scalar
    v2 g0, g1, de;
    float f0;
    {
        // donor from i-1 (geometry = x halves), own piece, donor from i+1 (y halves)
        const v2 E0m = (S[0].bc0 - refBC) + S[0].bc1 * bc(sD.x), E1m = S[0].bc1 * bc(bD.x);
        const v2 E0o = S[1].bc1 * bc(s1), E1o = S[1].bc1 * bc(b1);
        const v2 E0p = (S[2].bc0 - refBC) + S[2].bc1 * bc(sD.y), E1p = S[2].bc1 * bc(bD.y);
        const v2 J0m = E0m * bc(wD.x), J1m = E1m * bc(w2D.x);
        const v2 J0o = E0o * bc(w1), J1o = E1o * bc(w21);
        const v2 J0p = E0p * bc(wD.y), J1p = E1p * bc(w2D.y);
        g0 = (J0m + J0o) + J0p;
        g1 = (fma2(bc(xD.x), J0m, J1m) + fma2(bc(x1), J0o, J1o)) + fma2(bc(xD.y), J0p, J1p);
        de = fma2(bc(wD.x), S[0].de, fma2(bc(w1), S[1].de, S[2].de * bc(wD.y)));
        f0 = fmaf(wD.x, S[0].a2f.y, fmaf(w1, S[1].a2f.y, wD.y * S[2].a2f.y));
    }
    out[0] = ok ? refA + a0 : S[1].a01.x;
    out[1] = ok ? 12.0f * a1 : S[1].a01.y;
    out[2] = ok ? 180.0f * a2 : S[1].a2f.x;
    out[3] = ok ? refBC.x + g0.x : S[1].bc0.x;
    out[4] = ok ? 12.0f * g1.x : S[1].bc1.x;
    out[5] = ok ? refBC.y + g0.y : S[1].bc0.y;
    out[6] = ok ? 12.0f * g1.y : S[1].bc1.y;
    out[7] = ok ? de.x : S[1].de.x;
    out[8] = ok ? de.y : S[1].de.y;
    out[9] = ok ? f0 : S[1].a2f.y;
}

// =====================================================================================================
// NEXT-3 (reading R23): the confining sphere.  A cell whose centre lies outside the sphere is
// solid and never changes; along a pencil the fluid cells form one segment [lo, hi] whose ends are reflecting walls.
// The rings of the bulk path stay warp-uniform (whole brick records travel, solid cells included); what is per lane
// is only the image of the <= 4 ghost cells beyond each end of the lane's own segment, which are read straight from the
// input buffer (the mirror cells have long left, or not yet entered, the register windows), and the predicate on the store.
// =====================================================================================================
struct Segment { int lo, hi; };     // empty: lo > hi

// the oracle's criterion, operation by operation in fp64 with no contraction: ((X-cx)^2 + (Y-cy)^2) + (Z-cz)^2 > R^2
template <int DIR>
__device__ __forceinline__ bool sphere_inside(const SweepParams& P, double ta, double tb, int j) {
    const double xd = __dsub_rn(__dmul_rn((double)j + 0.5, P.sph_dx), P.sph_cd);
    const double dd = __dmul_rn(xd, xd);
    // ta, tb: squared offsets along the transverse axes a < b (in axis order); assemble in x, y, z order
    double sum;
    if (DIR == 0) sum = __dadd_rn(__dadd_rn(dd, ta), tb);
    else if (DIR == 1) sum = __dadd_rn(__dadd_rn(ta, dd), tb);
    else sum = __dadd_rn(__dadd_rn(ta, tb), dd);
    return !(sum > P.sph_r2);
}
template <int DIR>
__device__ __forceinline__ Segment sphere_segment(const SweepParams& P, int a, int b) {
    const double xa = __dsub_rn(__dmul_rn((double)a + 0.5, P.sph_dx), P.sph_ca), xb = __dsub_rn(__dmul_rn((double)b + 0.5, P.sph_dx), P.sph_cb);
    const double ta = __dmul_rn(xa, xa), tb = __dmul_rn(xb, xb);
    Segment sg; sg.lo = P.n; sg.hi = -1;
    // the inside set is an interval around the cell nearest the centre (every operation above is monotone in |x - c|)
    int seed = min(max((int)floor(P.sph_cd / P.sph_dx), 0), P.n - 1);
    if (!sphere_inside<DIR>(P, ta, tb, seed)) {
        if (seed + 1 < P.n && sphere_inside<DIR>(P, ta, tb, seed + 1)) seed += 1;
        else if (seed > 0 && sphere_inside<DIR>(P, ta, tb, seed - 1)) seed -= 1;
        else return sg;
    }
    const double h2 = P.sph_r2 - ta - tb;
    const int reach = h2 > 0.0 ? (int)(sqrt(h2) / P.sph_dx) : 0;
    int lo = max(seed - reach, 0), hi = min(seed + reach, P.n - 1);
    while (lo < seed && !sphere_inside<DIR>(P, ta, tb, lo)) ++lo;          // the estimate is within a cell or two
    while (lo > 0 && sphere_inside<DIR>(P, ta, tb, lo - 1)) --lo;
    while (hi > seed && !sphere_inside<DIR>(P, ta, tb, hi)) --hi;
    while (hi < P.n - 1 && sphere_inside<DIR>(P, ta, tb, hi + 1)) ++hi;
    sg.lo = lo; sg.hi = hi;
    return sg;
}
// image of cell index j / face index f under reflection at the segment's ends (again, if the segment is short)
__device__ __forceinline__ int fold_cell(const Segment& g, int j, float& sgn) {
    sgn = 1.0f;
#pragma unroll 1
    for (int it = 0; it < 16; ++it) {
        if (j < g.lo) { j = 2 * g.lo - 1 - j; sgn = -sgn; }
        else if (j > g.hi) { j = 2 * g.hi + 1 - j; sgn = -sgn; }
        else break;
    }
    return j;
}
__device__ __forceinline__ int fold_face(const Segment& g, int f) {
#pragma unroll 1
    for (int it = 0; it < 16; ++it) {
        if (f < g.lo) f = 2 * g.lo - f;
        else if (f > g.hi + 1) f = 2 * (g.hi + 1) - f;
        else break;
    }
    return f;
}

// =====================================================================================================
// The marching body, shared by every data path.  IO supplies plane n (hydro), cell n-3 (PPB coefficients,
// local family order, mirror signs applied) and takes the finished cell n-4.
// =====================================================================================================
// FLAT: 3-D flattening mode — the un-spread coefficient of cell n-2 is read from the detector field
// (pflat = the pencil's cell 0 in it) instead of being computed from the pencil's own pressures and velocities.
// CFL: S10 fused into the sweep — every finished cell folds max_d |u_d| + c of its NEW
// state into vmax, so that the step's last sweep leaves the next step's CFL maximum behind and ppm_cfl_dt has no pass
// of its own to make.
// SPH: confining sphere (above); seg = this lane's fluid segment, gpen = the lane's pencil in the INPUT buffer (cell 0, field 0).
// TWOF: two-fluid equation of state (reading R25): e = p beta(f), beta = beta2 + f dbeta with f the
// PPB cell mean clamped to [0,1]; Gamma = 1 + 1/beta of its own cell on each side of a face, the enthalpy flux with beta of the
// slab of gas the PPB remap donates through the face, the new pressure from the energy with beta of the NEW f.  mpen = the
// lane's pencil of m000 in the INPUT buffer (cell 0): Gamma of cell n-2 is needed one iteration before the rings hand over that
// cell's PPB coefficients, so m000 is read straight from global memory (an L2 hit: the bulk copy fetches the same lines), one
// iteration ahead of its use.
template <int DIR, int GRAV, bool FLAT, bool CFL, bool SPH, bool TWOF, class IO>
__device__ __forceinline__ void march(const SweepParams& P, IO& io, const int a, const int b, const int c0, const int c1,
                                      const bool valid, const unsigned wmask, const float* __restrict__ pflat, float& vmax,
                                      const Segment seg = Segment(), const float* __restrict__ gpen = nullptr,
                                      const float* __restrict__ mpen = nullptr) {
    const float gam = P.gamma, gp = P.gp, gmg = P.gmg, g_gm1 = P.g_gm1;
    const float dtdx = P.dtdx, hdt = P.hdt;

    Geo<DIR, GRAV> geo;
    geo.init(P, a, b);

    // sliding windows (registers).  q[s]: cell n-4+s
    V5 q[5];
    v2 fw[5];                                   // full (rho, p) of cells n-4 .. n
    v2 gi[4];                                   // slot s: (g of cell n-3+s, 1/rho of cell n-5+s) — two windows that shift together
    float g4 = 0.f;                             // g of cell n-4
#pragma unroll
    for (int s = 0; s < 5; ++s) { q[s] = zero5(); fw[s] = bc(1.f); }
#pragma unroll
    for (int s = 0; s < 4; ++s) gi[s] = mk(0.f, 1.f);
    V5 d2a = zero5(), d2b = zero5(), Fc = zero5(), Fcl = zero5(), parL = zero5(), parR = zero5();
    float WLr = 0.f, WLu = 0.f, WLp = 0.f, WLv = 0.f, WLw = 0.f;      // left state of the face being solved (from cell n-4)
    float Flm = 0.f, Fln = 0.f, FlE = 0.f;                              // fluxes through the left face of cell n-4
    v2 FlB = bc(0.f);
    float ft0 = 0.f, ft1 = 0.f, cs = 1.f;
    float ic2s = 1.f;                                                   // 1/c^2 of cell n-3
    v2 b0fc = bc(0.f);                                                  // (rho0, p0) at the face being solved
    PpbCell mw[3];
#pragma unroll
    for (int s = 0; s < 3; ++s) { mw[s].a01.x = mw[s].a01.y = mw[s].a2f.x = mw[s].a2f.y = 0.f; mw[s].bc0 = mw[s].bc1 = mw[s].de = bc(0.f); }
    int zw = 0;                                                         // which of the three cells of mw carry no higher PPB coefficient

    float fpre = 0.f;
    if (FLAT) {
        float sg;
        const int jf = image_cell(c0 - PPM_NGHOST - 2, P.n, P.bc_lo, P.bc_hi, sg);
        fpre = ld_flat(pflat + (long long)(jf >> 2) * P.FBd + ((jf & 3) << (2 * DIR)));
    }
    // two-fluid EOS: Gamma of cells n-4, n-3 (the cell n-2 joins them inside the iteration); m000 of cell n-2 in flight
    float Gm4 = gam, Gm3 = gam, mpre = 0.f;
    if (TWOF) {
        float sg;
        const int jf = image_cell(c0 - PPM_NGHOST - 2, P.n, P.bc_lo, P.bc_hi, sg);
        mpre = __ldg(mpen + (long long)(jf >> 2) * P.SBd + ((jf & 3) << (2 * DIR)));
    }
    // One iteration of the pipeline.  phase = integral_constant<int, S>:
    //   S = -1   any iteration: the brick phase n & 3, the boundary images and the pipeline-fill tests are run-time
    //   S = 0..3 an iteration of the steady state (bulk path only): n & 3 == S is a compile-time constant, every cell
    //            and face it touches lies inside the grid and the pipeline is full, so no image / fill logic remains
    auto body = [&](const int n, auto phase) {
        constexpr int S = decltype(phase)::value;
        io.template begin<S>(n);
        // ---- shift windows, take plane n ---------------------------------------------------------------
#pragma unroll
        for (int s = 0; s < 4; ++s) { q[s] = mv5(q[s + 1]); fw[s] = mv2(fw[s + 1]); }
        g4 = gi[0].x;
#pragma unroll
        for (int s = 0; s < 3; ++s) gi[s] = mv2(gi[s + 1]);
        float g_new;
        {
            float sgn, v[5];
            int j;
            io.template hydro<S>(n, j, sgn, v);
            if (SPH && (n < seg.lo || n > seg.hi) && n >= seg.lo - PPM_NGHOST && n <= seg.hi + PPM_NGHOST) {
                // a ghost cell of this lane's segment: the mirror image along the pencil, from the input buffer
                j = fold_cell(seg, n, sgn);
                const float* __restrict__ src = gpen + (long long)(j >> 2) * P.SBd + ((j & 3) << (2 * DIR));
                v[0] = __ldg(src);
                v[1] = sgn * __ldg(src + 64 * Dir<DIR>::U);
                v[2] = __ldg(src + 64 * Dir<DIR>::V);
                v[3] = __ldg(src + 64 * Dir<DIR>::W);
                v[4] = __ldg(src + 64 * 4);
            }
            q[4].A = mk(v[0], v[4]); q[4].B = mk(v[2], v[3]); q[4].u = v[1];
            const Base bs = geo.cell(P, j, sgn);
            fw[4] = bs.rp + q[4].A;
            g_new = bs.g;
        }
        // ---- E, F: flattening ---------------------------------------------------------------------------
        // 1/rho is taken once per cell and carried (the tracing and the PPB masses need it again), and c and 1/c^2 come
        // from ONE reciprocal square root: c = x rsqrt(x), 1/c^2 = rsqrt(x)^2 with x = gamma p / rho
        gi[3] = mk(g_new, rcp(fw[2].x));
        float Gm2 = gam;                                             // adiabatic index of cell n-2
        if (TWOF) {
            Gm2 = 1.0f + rcp(fmaf(sat(mpre), P.dbeta, P.beta2));     // Gamma = 1 + 1/beta(f), f = m000 clamped to [0,1]
            float sg;
            const int jf = (S >= 0) ? n - 1 : image_cell(n - 1, P.n, P.bc_lo, P.bc_hi, sg);     // (m000 is even under the mirror)
            mpre = __ldg(mpen + (long long)(jf >> 2) * P.SBd + ((jf & 3) << (2 * DIR)));
        }
        const float xc = Gm2 * fw[2].y * gi[3].y;
        const float icn = rsqrtf(fmaxf(xc, 1e-37f));
        const float cn2 = xc * icn;                                  // c_{n-2}
        const float ic2n = icn * icn;
        float ftn;
        if (FLAT) {
            ftn = fpre;                                              // F~_{n-2}, in flight since the last iteration
            float sg;
            const int jf = (S >= 0) ? n - 1 : image_cell(n - 1, P.n, P.bc_lo, P.bc_hi, sg);     // (the detector is mirror-invariant)
            fpre = ld_flat(pflat + (long long)(jf >> 2) * P.FBd + ((jf & 3) << (2 * DIR)));
        } else {
            // The jump ramp clamp(3|d1|/min(p) - 1) is zero wherever the pressure changes by less than a third over two
            // cells: everywhere but in strong shocks.  When no lane of the warp is near one, f~ = 0 without the three
            // divisions (a warp-uniform shortcut: the result is the same zero the ramps would give).
            const float d1 = fw[3].y - fw[1].y;
            const float pm = fminf(fw[3].y, fw[1].y);
            ftn = 0.f;
            if (!(PPM_UNIFORM_FAST & 1) || !__all_sync(wmask, 3.0f * fabsf(d1) <= pm || !valid)) {
                const float dd2 = fw[4].y - fw[0].y;
                const float steep = sat(10.0f * (fdiv(fabsf(d1), fmaxf(fabsf(dd2), PPM_TINY)) - 0.75f));
                const float jump = sat(fdiv(3.0f * fabsf(d1), pm) - 1.0f);
                const float conv = sat(fdiv(q[1].u - q[3].u, 0.05f * cn2));
                ftn = steep * jump * conv;
            }
        }
        const float fl3 = fmaxf(ft0, fmaxf(ft1, ftn));              // f_{n-3}
        // no flattening anywhere in the warp (every smooth flow): the parabola is used as it is — f (q - L) + L with
        // f = 0 is L bit for bit, so skipping the blend changes nothing
        const bool noflat = (PPM_UNIFORM_FAST & 1) && __all_sync(wmask, fl3 == 0.f || !valid);
        // ---- G, H: flattened parabola and characteristic tracing of cell n-3 ---------------------------
        // Each traced quantity is a pair W = (left of face (n-3)+1/2, right of face (n-3)-1/2): the two states
        // are mirror images, F+ and F- differ only in the sign of the q6 term.
        v2 Wr, Wu, Wp, Wv, Ww;
        v2 b0fn;
        {
            int fi = (S >= 0) ? n - 2 : image_face(n - 2, P.n, P.bc_lo, P.bc_hi);
            if (SPH && (n - 2 < seg.lo || n - 2 > seg.hi + 1) && seg.lo <= seg.hi) fi = fold_face(seg, n - 2);
            b0fn = geo.face(P, fi);
        }
        {
            const V5 qc = q[1];
            V5 L = parL, R = parR;
            if (!noflat) {
                L = fma5(qc - parL, fl3, parL);
                R = fma5(qc - parR, fl3, parR);
            }
            const V5 dq = R - L;
            const V5 q6 = fma5(L + R, -3.0f, qc * 6.0f);
            const float rho = fw[1].x, c = cs, u = qc.u;
            const float c2 = c * c, rc = rho * c, ic2 = ic2s, ic2h = 0.5f * ic2, cor = c * gi[2].y;
            const float s_m = (u - c) * dtdx, s_0 = u * dtdx, s_p = (u + c) * dtdx;
            // Each wave family k takes its amplitude from its own domain of dependence max(+-sigma^k, 0); a
            // wave moving away from the face has the zero-width domain, i.e. the edge value (reading R8',
            // DESIGN.md).  No switch on sign(lambda^k): the traced states are continuous in the data.
            // domains (left state, right state): fastest wave toward the face, the opposite acoustic wave, the entropy wave
            const v2 sf = mk(fmaxf(s_p, 0.f), fmaxf(-s_m, 0.f));
            const v2 so = mk(fmaxf(s_m, 0.f), fmaxf(-s_p, 0.f));
            const v2 se = mk(fmaxf(s_0, 0.f), fmaxf(-s_0, 0.f));
            // H5: A(s) = (s/2) (dq -+ (1 - 2s/3) q6)   (- for the left state = qR - F+, + for the right = F- - qL)
            const v2 K23 = mk(2.0f / 3.0f, -2.0f / 3.0f), Km1 = mk(-1.0f, 1.0f);
            const v2 hf = sf * 0.5f, tf = fma2(sf, K23, Km1);
            const v2 ho = so * 0.5f, to = fma2(so, K23, Km1);
            const v2 he = se * 0.5f, te = fma2(se, K23, Km1);
#define PPM_AV(dq_, q6_, h_, t_) ((h_) * fma2((t_), bc(q6_), bc(dq_)))
            const v2 Ar = PPM_AV(dq.A.x, q6.A.x, hf, tf), Au = PPM_AV(dq.u, q6.u, hf, tf), Ap = PPM_AV(dq.A.y, q6.A.y, hf, tf);
            const v2 Ou = PPM_AV(dq.u, q6.u, ho, to), Op = PPM_AV(dq.A.y, q6.A.y, ho, to);
            const v2 Er = PPM_AV(dq.A.x, q6.A.x, he, te), Ep = PPM_AV(dq.A.y, q6.A.y, he, te);
            const v2 Ev = PPM_AV(dq.B.x, q6.B.x, he, te), Ew = PPM_AV(dq.B.y, q6.B.y, he, te);
#undef PPM_AV
            // acoustic amplitude of the opposite family: beta = (am, -ap);  entropy amplitude al0 = (a0L, -a0R)
            const v2 du = Ou - Au, dp = Op - Ap;
            const v2 beta = fma2(np(du), bc(rc), dp) * ic2h;
            const v2 al0 = fma2(Ep - Ap, bc(-ic2), Er - Ar);
            // W = (qR, qL) + (-,+) * (...)
            const v2 K10 = PPM_K10_PARAM ? up(P.k10) : mk(1.0f, 0.0f);      // (1, 0): as a 64-bit kernel argument it sits in a uniform register pair
            const v2 Br = fma2(bc(dq.A.x), K10, bc(L.A.x)), Bu = fma2(bc(dq.u), K10, bc(L.u)), Bp = fma2(bc(dq.A.y), K10, bc(L.A.y));
            const v2 Bv = fma2(bc(dq.B.x), K10, bc(L.B.x)), Bw = fma2(bc(dq.B.y), K10, bc(L.B.y));
            Wr = Br + np((Ar + beta) + al0);
            Wu = (Bu + np(Au)) + beta * cor;
            Wp = Bp + np(fma2(beta, bc(c2), Ap));
            Wv = Bv + np(Ev);
            Ww = Bw + np(Ew);
            if (GRAV != PPM_GRAV_NONE) {   // half-step sources of the perturbation equations (H6)
                const v2 db = b0fn - b0fc;
                const float k = -hdt * u * P.inv_dx;
                const float su = hdt * gi[0].x * (qc.A.x * gi[2].y);
                Wr = Wr + bc(k * db.x); Wp = Wp + bc(k * db.y); Wu = Wu + bc(su);
            }
        }
        // ---- A, B, C, D: interpolation of cell n-2 (placed after the tracing of cell n-3, the last reader of the carried
        //      parabola: the new one can then take its registers and the rotation at the loop end costs no move) ----
        const V5 d2n = fma5(q[3], -2.0f, q[4]) + q[2];                                           // d2_{n-1}
        const V5 Fn = fma5(q[1] + q[4], -1.0f / 12.0f, (q[2] + q[3]) * (7.0f / 12.0f));          // face (n-2)+1/2 (H1)
        const V5 Fnl = map3(q[2], Fn, q[3], [](float x, float y, float z) { return med3(x, y, z); });   // H2: clamp
        V5 pLn, pRn;
        {
            const V5 num = d2n - d2a;
            const V5 den = fma5(abs5(d2b), 2.0f, abs5(d2a)) + (abs5(d2n) + bc5(PPM_TINY));
            const V5 om = map3(num, den, den, [](float x, float y, float) { return sat(fmaf(fabsf(x) * rcp(y), 5.0f, -0.5f)); });   // H3
            parabola(q[2], Fcl, Fnl, Fc, Fn, om, pLn, pRn);
        }
        // ---- K (first half): PPB coefficients of cell n-3, pre-limited (P2) ---------------------------
        // (two-fluid mode takes them BEFORE the Riemann problem: its energy flux needs the donor cells' polynomials)
        auto ppb_take = [&]() {
        mv_ppb(mw[0], mw[1]); mv_ppb(mw[1], mw[2]);
        if (S >= 0 || n - 3 >= c0 - 1) {
            float m[10];
            io.template ppb<S>(n - 3, m);
            if (SPH && (n - 3 < seg.lo || n - 3 > seg.hi) && n - 3 >= seg.lo - PPM_NGHOST && n - 3 <= seg.hi + PPM_NGHOST) {
                float sg;
                const int j = fold_cell(seg, n - 3, sg);
                const float* __restrict__ src = gpen + (long long)(j >> 2) * P.SBd + ((j & 3) << (2 * DIR));
#pragma unroll
                for (int k = 0; k < 10; ++k) m[k] = __ldg(src + 64 * (5 + PPB_PERM[DIR][k]));
                m[1] *= sg; m[4] *= sg; m[6] *= sg;            // the coefficients odd in the normal direction
            }
            // bound B: first-order terms 1/2, pure second-order 1/6, mixed 1/4.
            // local order: a1,b0,c0 are P1 terms; a2,d0,e0 are P2 terms; b1,c1,f0 are mixed P1P1 terms.
            const v2 bc0 = mk(m[3], m[5]), bc1 = mk(m[4], m[6]), de = mk(m[7], m[8]);
            const v2 Bp = fma2(abs2(bc1), bc(0.25f), fma2(abs2(de), bc(1.0f / 6.0f), abs2(bc0) * 0.5f));
            const float B = fmaf(fabsf(m[9]), 0.25f, fmaf(fabsf(m[2]), 1.0f / 6.0f, fmaf(fabsf(m[1]), 0.5f, hsum(Bp))));
            // theta = min(1, max(0, min(m000, 1 - m000)) / B): 1 wherever the bound B already fits (the constraint is
            // "almost never performed") — then the coefficients are taken as they are
            const float room = fmaxf(0.f, fminf(m[0], 1.0f - m[0]));
            // (a real copy: the register m[0] arrived in is about to be reloaded by the prefetch below)
            if (IO::HAS_FAST) mw[2].a01.x = m[0];
            else asm volatile("mov.f32 %0, %1;" : "=f"(mw[2].a01.x) : "f"(m[0]));
            if ((PPM_UNIFORM_FAST & 8) && __all_sync(wmask, B <= room || !valid)) {
                mw[2].a01.y = m[1]; mw[2].a2f.x = m[2]; mw[2].a2f.y = m[9];
                mw[2].bc0 = bc0; mw[2].bc1 = bc1; mw[2].de = de;
            } else {
                const float th = (B <= room) ? 1.0f : fdiv(room, fmaxf(B, PPM_TINY));
                mw[2].a01.y = m[1] * th; mw[2].a2f.x = m[2] * th; mw[2].a2f.y = m[9] * th;
                mw[2].bc0 = bc0 * th; mw[2].bc1 = bc1 * th; mw[2].de = de * th;
            }
            io.ppb_prefetch(n - 2, mw[2]);   // one cell ahead of its use (overshoots by one at the end: still a valid image cell)
            // bit s of zw: the nine higher coefficients of cell n-5+s all vanish (B is a positive combination of their moduli)
            if (PPM_FV_SKIP) zw = ((zw << 1) | ((B == 0.f && P.fv_shortcut) ? 1 : 0)) & 7;       // (the run-time switch is folded in here: no branch of its own)
        } else if (PPM_FV_SKIP) zw = (zw << 1) & 7;
        };
        if (TWOF) ppb_take();
        // ---- I: Riemann problem at face (n-4)+1/2 : L = left state carried from cell n-4, R = right state of cell n-3
        float Frm, Frn, FrE;
        v2 FrB;
        {
            const float r0f = b0fc.x, p0f = b0fc.y;
            const float pfl = P.p_floor - p0f;
            const v2 Zu = mk(WLu, Wu.y);
            v2 r = bc(r0f) + mk(WLr, Wr.y);
            r = mk(fmaxf(r.x, P.rho_floor), fmaxf(r.y, P.rho_floor));
            const v2 pp = mk(fmaxf(WLp, pfl), fmaxf(Wp.y, pfl));              // p' (floored)
            const v2 p = bc(p0f) + pp;
            const v2 GK2 = mk(Gm4, Gm3);                                       // two-fluid: Gamma of the left cell n-4, of the right cell n-3
            const v2 C2 = TWOF ? (p * GK2) * r : (p * gam) * r;
            const v2 C = C2 * mk(rsqrtf(fmaxf(C2.x, 1e-37f)), rsqrtf(fmaxf(C2.y, 1e-37f)));
            const float CLR = C.x * C.y;
            float pps = fmaxf(pfl, fdiv(hsum(swp(C) * pp) + CLR * (Zu.x - Zu.y), C.x + C.y));   // p*' acoustic guess
            // W_K^2 = rho_K ((G+1)/2 p* + (G-1)/2 p_K) = gpr p* + gmr
            const v2 gpr = TWOF ? r * fma2(GK2, bc(0.5f), bc(0.5f)) : r * gp;
            const v2 gmr = TWOF ? (p * r) * fma2(GK2, bc(0.5f), bc(-0.5f)) : C2 * gmg;
            // Newton on p*' with the two-shock wave speeds W_K; at most 5 iterations (reading R7).  The loop
            // stops early only when EVERY lane's last update is below fp32 resolution of p* (warp-uniform
            // exit), i.e. when further iterations could not change the result beyond rounding.
            v2 w2, iw;                                                        // W_K^2 and 1/W_K of the latest iteration
            auto newton = [&]() -> bool {
                const float ps = p0f + pps;
                w2 = fma2(gpr, bc(ps), gmr);
                iw = mk(rsqrtf(w2.x), rsqrtf(w2.y));
                const v2 us = fma2(np(bc(pps) - pp), iw, Zu);               // u*_L = uL - (p*-pL)/W_L, u*_R = uR + (p*-pR)/W_R
                const v2 iz = (w2 + C2) * ((iw * iw) * iw);                   // 1/Z_K = (W^2 + C^2) / (2 W^3), times 2
                const float d = fdiv(2.0f * (us.y - us.x), hsum(iz));
                pps = fmaxf(pfl, pps - d);
                return fabsf(d) <= 6e-8f * ps;
            };
            // first iteration in straight-line code (the scheduler can overlap it with independent work); the
            // remaining ones only while some lane still moves (rare at low Mach: the acoustic guess is nearly exact)
            // (lanes on pad cells of a ragged grid carry garbage and do not vote)
            bool conv = __all_sync(wmask, newton() || !valid);
#if PPM_NEWTON_NESTED
            // (nested rather than looped: a loop makes ptxas copy a dozen operands into the loop's registers on every pass
            // through here, though the loop body itself runs for strong shocks only)
            if (!conv) { conv = __all_sync(wmask, newton() || !valid);
                if (!conv) { conv = __all_sync(wmask, newton() || !valid);
                    if (!conv) { conv = __all_sync(wmask, newton() || !valid);
                        if (!conv) conv = __all_sync(wmask, newton() || !valid); } } }
#else
            if (!conv) {
#pragma unroll 1
                for (int it = 1; it < 5; ++it)
                    if ((conv = __all_sync(wmask, newton() || !valid))) break;
            }
#endif
            const float ps = p0f + pps;
            // "then recompute W_K" at the final p* (H7).  After a converged iteration p* moved by less than one fp32
            // rounding of itself, so W_K of that iteration IS W_K(p*) to rounding: it is reused.  Only when the
            // iteration cap ended the loop (strong shocks) is it evaluated again.
            if (!(PPM_UNIFORM_FAST & 2) || !conv) {
                w2 = fma2(gpr, bc(ps), gmr);
                iw = mk(rsqrtf(fmaxf(w2.x, 1e-37f)), rsqrtf(fmaxf(w2.y, 1e-37f)));
            }
            const v2 Ws = w2 * iw;
            const float us = fdiv(hsum(Ws * Zu) + (pp.x - pp.y), hsum(Ws));
            // sampling at x/t = 0 in the frame mirrored so that the upwind side K is on the left
            const bool left = us >= 0.f;
            const float sg = left ? 1.f : -1.f;
            const float rK = left ? r.x : r.y, uK = left ? Zu.x : Zu.y, pK = left ? p.x : p.y, ppK = left ? pp.x : pp.y;
            const float wk2 = left ? w2.x : w2.y, WK = left ? Ws.x : Ws.y;
            const v2 vw = mk(left ? WLv : Wv.y, left ? WLw : Ww.y);
            const float GK = TWOF ? (left ? Gm4 : Gm3) : gam;                  // the gas on the upwind side of the contact
            float rs = fdiv(rK * wk2, wk2 - rK * (pps - ppK));                 // 1/(1/rK - (p*-pK)/WK^2)
            rs = fmaxf(rs, P.rho_floor);
            const float uKh = sg * uK, ush = sg * us;
            const bool shock = pps > ppK;
            // The face lies in the star region (theta = 1) when the upwind wave runs upwind: a shock with
            // u_K - W_K/rho_K < 0, or a fan whose head u_K - c_K AND tail u* - c*_K are negative — every face of a
            // subsonic flow.  Written without the two sound speeds (u^2 rho < gamma p), and when it holds for every lane
            // of the warp the sampled state is the star state itself.
            const bool star = shock ? (uKh * rK < WK) : ((uKh < 0.f || uKh * uKh * rK < GK * pK) && ush * ush * rs <= GK * ps);
            float rh = rs, uh = us, pph = pps;
            if (!(PPM_UNIFORM_FAST & 4) || !__all_sync(wmask, star || !valid)) {
                const float irK = rcp(rK);
                const float cK = fsqrt(GK * pK * irK), cst = fsqrt(GK * ps * rcp(rs));
                const float lam_head = uKh - (shock ? WK * irK : cK);
                const float lam_tail = shock ? lam_head : ush - cst;
                const float th = (lam_head >= 0.f) ? 0.f : ((lam_tail <= 0.f) ? 1.f : fdiv(-lam_head, lam_tail - lam_head));
                rh = fmaf(th, rs - rK, rK);
                uh = fmaf(th, us - uK, uK);
                pph = fmaf(th, pps - ppK, ppK);
            }
            const float ph = p0f + pph;
            const float Fm = rh * uh;
            Frm = Fm;
            Frn = fmaf(Fm, uh, pph);
            FrB = vw * Fm;
            if (TWOF) {
                // the enthalpy of the gas that crosses the face: beta of the mean FV of the slab of mass dt Fm that the PPB
                // remap takes out of the donor cell (its pre-limited polynomial along the sweep; reading R25)
                const bool fwd = Fm >= 0.f;
                const float da0 = fwd ? mw[1].a01.x : mw[2].a01.x, da1 = fwd ? mw[1].a01.y : mw[2].a01.y, da2 = fwd ? mw[1].a2f.x : mw[2].a2f.x;
                const float sig = fminf(dtdx * fabsf(Fm) * (fwd ? gi[1].y : gi[2].y), 1.0f);       // donated fraction of the donor's mass
                const float hs = fmaf(-0.5f, sig, 0.5f), sm = fwd ? hs : -hs;                       // slab midpoint in its mass coordinate
                const float fs = fmaf(da2, fmaf(sm, sm, fmaf(sig * sig, 1.0f / 12.0f, -1.0f / 12.0f)), fmaf(da1, sm, da0));
                const float bt1 = fmaf(sat(fs), P.dbeta, P.beta2) + 1.0f;
                FrE = uh * fmaf(bt1, ph, 0.5f * rh * fmaf(uh, uh, hsum(vw * vw)));
            } else
            FrE = uh * fmaf(g_gm1, ph, 0.5f * rh * fmaf(uh, uh, hsum(vw * vw)));
        }
        if (!TWOF) ppb_take();
        // ---- J, K, L: finish cell n-4 ---------------------------------------------------------------------
        const int i = n - PPM_NGHOST;
        if (S >= 0 || i >= c0) {
            // the cell's old values: the bulk path still has them in shared memory (its results overwrite them below),
            // so the register window need not carry them for four iterations
            V5 qo = q[0];
            if (IO::HAS_OLD) {
                float v[5];
                io.template old_hydro<S>(i, v);
                qo.A = mk(v[0], v[4]); qo.B = mk(v[2], v[3]); qo.u = v[1];
            }
            const float r_old = fw[0].x, rp_old = qo.A.x, pp_old = qo.A.y, u0 = qo.u, g = g4;
            const v2 vw0 = qo.B;
            float drho = -dtdx * (Frm - Flm);
            int bad = 0;
            if (!(r_old + drho > P.rho_floor)) { drho = P.rho_floor - r_old; bad = 1; }
            const float r_new = r_old + drho;
            const float rp_new = rp_old + drho;
            const float mu0 = r_old * u0;
            float mu1 = mu0 - dtdx * (Frn - Fln);
            float dE = -dtdx * (FrE - FlE);
            if (GRAV != PPM_GRAV_NONE) {
                mu1 += P.dt * 0.5f * (rp_old + rp_new) * g;
                dE += P.dt * 0.5f * (mu0 + mu1) * g;
            }
            const v2 mB = fma2(FrB - FlB, bc(-dtdx), vw0 * r_old);
            const float irn = rcp(r_new);
            float ho[5], mo[10];
            const float u1 = mu1 * irn;
            const v2 vw1 = mB * irn;
            const float dKE = 0.5f * (r_new * fmaf(u1, u1, hsum(vw1 * vw1)) - r_old * fmaf(u0, u0, hsum(vw0 * vw0)));
            float pp_new, Gnew = gam;
            if (TWOF) {
                // p beta is what the energy equation advances: p_new = (p_old beta_old + dE - dKE) / beta_new with beta of the
                // NEW cell mean of FV, i.e. after this sweep's remap; in increment form on the perturbation
                // (the uniform-FV shortcut, see below: the remap returns the cell's own mean and nine zeros)
                const bool fvu2 = PPM_FV_SKIP && __all_sync(wmask, (zw == 7 && mw[0].a01.x == mw[1].a01.x && mw[1].a01.x == mw[2].a01.x) || !valid);
                if (fvu2) {
                    mo[0] = mw[1].a01.x;
#pragma unroll
                    for (int k = 1; k < 10; ++k) mo[k] = 0.f;
                } else ppb_remap<false>(mw, gi[0].y, gi[1].y, gi[2].y, r_new, irn, dtdx * Flm, dtdx * Frm, mo);
                const float ibn = rcp(fmaf(sat(mo[0]), P.dbeta, P.beta2));
                pp_new = pp_old + ((dE - dKE) - fw[0].y * (P.dbeta * (sat(mo[0]) - sat(mw[1].a01.x)))) * ibn;
                Gnew = 1.0f + ibn;
            } else pp_new = pp_old + (gam - 1.0f) * (dE - dKE);
            const float p0c = fw[0].y - pp_old;
            if (!(p0c + pp_new > P.p_floor)) { pp_new = P.p_floor - p0c; bad = 1; }
            const bool fluid = !SPH || (i >= seg.lo && i <= seg.hi);
            if (bad && valid && fluid) atomicOr(P.flag, (r_new == r_new && pp_new == pp_new) ? 1 : 2);
            if (CFL && fluid) {                                         // C6 on the new state: c from the full rho, p
                const float xs = Gnew * (p0c + pp_new) * irn;
                const float cnew = xs * rsqrtf(fmaxf(xs, 1e-37f));
                vmax = fmaxf(vmax, fmaxf(fabsf(u1), fmaxf(fabsf(vw1.x), fabsf(vw1.y))) + cnew);
            }
            ho[0] = rp_new; ho[1] = u1; ho[2] = vw1.x; ho[3] = vw1.y; ho[4] = pp_new;
            if (!TWOF) {
                // Where FV is uniform — the three cells the remap draws from have the same mean and no higher coefficient, in every
                // pencil of the warp — the remap returns that mean and nine zeros whatever mass moves (every piece integrates a
                // deviation from the own cell's constant that is identically zero): the same values, without the ~120 instructions.
                // (Most of a star: the tracked gas differs from its surroundings only near the boundary of the convection zone.)
                const bool fvu = PPM_FV_SKIP && __all_sync(wmask, (zw == 7 && mw[0].a01.x == mw[1].a01.x && mw[1].a01.x == mw[2].a01.x) || !valid);
                if (fvu) {
                    mo[0] = mw[1].a01.x;
#pragma unroll
                    for (int k = 1; k < 10; ++k) mo[k] = 0.f;
                } else ppb_remap<false>(mw, gi[0].y, gi[1].y, gi[2].y, r_new, irn, dtdx * Flm, dtdx * Frm, mo);
            }
            io.template store<S>(i, ho, mo, fluid);
        }
        // ---- rotate the carried pipeline registers ----------------------------------------------------
        d2a = mv5(d2b); d2b = MV5B(d2n); Fc = MV5B(Fn); Fcl = MV5B(Fnl); parL = MV5C(pLn); parR = MV5C(pRn);
        WLr = Wr.x; WLu = Wu.x; WLp = Wp.x; WLv = Wv.x; WLw = Ww.x;
        Flm = Frm; Fln = Frn; FlE = FrE; FlB = MV2D(FrB);
        ft0 = ft1; ft1 = ftn; cs = cn2; b0fc = b0fn;
        ic2s = ic2n;
        if (TWOF) { Gm4 = Gm3; Gm3 = Gm2; }
    };
    using std::integral_constant;
    if (IO::HAS_FAST) {
        // bulk path: c0, c1 are multiples of 4.  Ghost bricks and pipeline fill [c0 - 4, c0 + 4) and the drain
        // [c1, c1 + 4) run the generic body (ONE copy of it: the two passes of the outer loop); the bricks in between
        // run the steady-state body, unrolled over the four cells of a brick — the sliding windows become register
        // renaming and the brick-phase logic constant-folds.
#pragma unroll 1
        for (int pass = 0; pass < 2; ++pass) {
            const int lo = pass ? c1 : c0 - PPM_NGHOST, hi = pass ? c1 + PPM_NGHOST : c0 + 4;
#pragma unroll 1
            for (int n = lo; n < hi; ++n) body(n, integral_constant<int, -1>());
            if (pass == 0) {
#if PPM_FAST_UNROLL == 4
#pragma unroll 1
                for (int n = c0 + 4; n < c1; n += 4) {
                    body(n, integral_constant<int, 0>());
                    body(n + 1, integral_constant<int, 1>());
                    body(n + 2, integral_constant<int, 2>());
                    body(n + 3, integral_constant<int, 3>());
                }
#elif PPM_FAST_UNROLL == 2
#pragma unroll 1
                for (int n = c0 + 4; n < c1; n += 2) {
                    body(n, integral_constant<int, 4>());
                    body(n + 1, integral_constant<int, 5>());       // (a second type, so that the body is inlined twice)
                }
#else
#pragma unroll 1
                for (int n = c0 + 4; n < c1; ++n) body(n, integral_constant<int, 4>());
#endif
            }
        }
    } else {
#pragma unroll MARCH_UNROLL
        for (int n = c0 - PPM_NGHOST; n < c1 + PPM_NGHOST; ++n) body(n, integral_constant<int, -1>());
    }
    io.finish();
}

// =====================================================================================================
// NEXT-2 (Fig. 3): PPB-only sweep.  The hydro state is held fixed (direct path: its fields are
// copied through; bulk-staged path: they stay in their buffer, see IoBulk<DIR, ADV>) and FV is advected by the stored velocity field: uniform gas (rho = 1), face velocity = mean of
// the two cell values, mass through the face = dt * u_f (reading R22); P2-P4 exactly as in march().
// Same iteration timing as march(), so the IO classes serve both: iteration n takes the velocity of cell n and
// the coefficients of cell n-3, and finishes cell n-4.
// =====================================================================================================
template <int DIR, class IO>
__device__ __forceinline__ void march_ppb(const SweepParams& P, IO& io, const int c0, const int c1) {
    const float dtdx = P.dtdx;
    float uw[5] = {0.f, 0.f, 0.f, 0.f, 0.f};                // normal velocity of cells n-4 .. n
    float Flm = 0.f;                                        // u at the left face of cell n-4
    PpbCell mw[3];
#pragma unroll
    for (int s = 0; s < 3; ++s) { mw[s].a01.x = mw[s].a01.y = mw[s].a2f.x = mw[s].a2f.y = 0.f; mw[s].bc0 = mw[s].bc1 = mw[s].de = bc(0.f); }
#pragma unroll 1
    for (int n = c0 - PPM_NGHOST; n < c1 + PPM_NGHOST; ++n) {
        io.template begin<-1>(n);
#pragma unroll
        for (int s = 0; s < 4; ++s) uw[s] = uw[s + 1];
        {
            float sgn, v[5];
            int j;
            io.template hydro<-1>(n, j, sgn, v);
            uw[4] = v[1];
        }
        const float Frm = 0.5f * (uw[0] + uw[1]);           // face (n-4)+1/2
        mw[0] = mw[1]; mw[1] = mw[2];
        if (n - 3 >= c0 - 1) {
            float m[10];
            io.template ppb<-1>(n - 3, m);
            const v2 bc0 = mk(m[3], m[5]), bc1 = mk(m[4], m[6]), de = mk(m[7], m[8]);
            const v2 Bp = fma2(abs2(bc1), bc(0.25f), fma2(abs2(de), bc(1.0f / 6.0f), abs2(bc0) * 0.5f));
            const float B = fmaf(fabsf(m[9]), 0.25f, fmaf(fabsf(m[2]), 1.0f / 6.0f, fmaf(fabsf(m[1]), 0.5f, hsum(Bp))));
            const float th = fminf(1.0f, fdiv(fmaxf(0.f, fminf(m[0], 1.0f - m[0])), fmaxf(B, PPM_TINY)));
            asm volatile("mov.f32 %0, %1;" : "=f"(mw[2].a01.x) : "f"(m[0]));
            mw[2].a01.y = m[1] * th; mw[2].a2f.x = m[2] * th; mw[2].a2f.y = m[9] * th;
            mw[2].bc0 = bc0 * th; mw[2].bc1 = bc1 * th; mw[2].de = de * th;
            io.ppb_prefetch(n - 2, mw[2]);
        }
        const int i = n - PPM_NGHOST;
        if (i >= c0) {
            float mo[10];
            const float rn = 1.0f - dtdx * (Frm - Flm);
            ppb_remap<true>(mw, 1.0f, 1.0f, 1.0f, rn, rcp(fmaxf(rn, PPM_TINY)), dtdx * Flm, dtdx * Frm, mo);
            io.template store_ppb<-1>(i, mo);
        }
        Flm = Frm;
    }
    io.finish();
}

// =====================================================================================================
// IoDirect: straight global loads / stores.  16 lanes = the 4x4 pencils of one brick column; a load of one
// field is one 64-byte brick layer per half warp.  A cell's 15 fields sit 256 B apart in its brick record, so
// each of the three access streams (hydro plane n+1, PPB cell n-2, finished cell n-4) needs one pointer per
// iteration and the fields are compile-time offsets.  Next plane / next PPB cell prefetched into registers.
// =====================================================================================================
template <int DIR>
struct IoDirect {
    static constexpr bool HAS_OLD = false;   // no staged copy of a cell's old values: march() carries them in registers
    static constexpr bool HAS_FAST = false;  // no steady-state body: any extent, any segment bounds
    template <int S> __device__ __forceinline__ void old_hydro(int, float (&)[5]) {}
    static constexpr int SH = 2 * DIR;       // in-brick stride along the sweep axis = 1 << SH floats
    const SweepParams& P;
    const float* __restrict__ const pin;     // the thread's pencil: cell 0 of the sweep axis, field 0
    float* __restrict__ const pout;
    float nx5[5];            // plane n+1, already in flight
    float nm[10];            // PPB coefficients of the next cell, already in flight
    int jn; float sn, snm;
    __device__ __forceinline__ IoDirect(const SweepParams& P_, long long tb, int n0, int c0) : P(P_), pin(P_.in + tb), pout(P_.out + tb) { fetch(n0); fetch_ppb(c0 - 1); }
    // float offset of cell j along the pencil (same for every lane)
    __device__ __forceinline__ long long off(int j) const { return (long long)(j >> 2) * P.SBd + ((j & 3) << SH); }
    __device__ __forceinline__ void fetch(int n) {
        jn = image_cell(n, P.n, P.bc_lo, P.bc_hi, sn);
        const float* __restrict__ p = pin + off(jn);
        if (PPM_PREFETCH_BRICKS > 0 && (n & 3) == 0 && (unsigned)(n + 4 * PPM_PREFETCH_BRICKS) < (unsigned)P.n) {
            // first plane of a brick: ask L2 for the record PPM_PREFETCH_BRICKS further along (3840 contiguous bytes,
            // one request per brick column = per half warp); also walks the TLB ahead of the loads
            if ((threadIdx.x & 15) == 0)
                asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(pin + off(n + 4 * PPM_PREFETCH_BRICKS)), "n"(PPM_BRICK_FLOATS * 4) : "memory");
        }
        nx5[0] = __ldg(p);
        nx5[1] = __ldg(p + 64 * Dir<DIR>::U);
        nx5[2] = __ldg(p + 64 * Dir<DIR>::V);
        nx5[3] = __ldg(p + 64 * Dir<DIR>::W);
        nx5[4] = __ldg(p + 64 * 4);
    }
    template <int S> __device__ __forceinline__ void begin(int) {}
    template <int S> __device__ __forceinline__ void hydro(int n, int& j, float& sgn, float (&v)[5]) {
        j = jn; sgn = sn;
#pragma unroll
        for (int k = 0; k < 5; ++k) v[k] = nx5[k];
        v[1] *= sgn;
        fetch(n + 1);        // overshoots by one plane at the end of the pencil: still a valid image cell
    }
    __device__ __forceinline__ void fetch_ppb(int c) {
        const int j = image_cell(c, P.n, P.bc_lo, P.bc_hi, snm);
        const float* __restrict__ p = pin + off(j);
#pragma unroll
        for (int k = 0; k < 10; ++k) nm[k] = __ldg(p + 64 * (5 + PPB_PERM[DIR][k]));
    }
    template <int S> __device__ __forceinline__ void ppb(int, float (&m)[10]) {
#pragma unroll
        for (int k = 0; k < 10; ++k) m[k] = nm[k];
        m[1] *= snm; m[4] *= snm; m[6] *= snm;
    }
    // Issues the loads of cell c one iteration ahead of their use.  `used` = the values computed from the
    // previous prefetch: the empty asm orders the new loads after them, so the loads land in the very
    // registers the old values just left (otherwise ptxas hoists the loads above the last use, renames them,
    // and parks a register copy — which waits for DRAM — right behind the loads).
    __device__ __forceinline__ void ppb_prefetch(int c, const PpbCell& used) {
        const int j = image_cell(c, P.n, P.bc_lo, P.bc_hi, snm);
        const float* p = pin + off(j);
        asm volatile("" : "+l"(p) : "f"(used.a01.x), "f"(used.a01.y), "f"(used.a2f.x), "f"(used.a2f.y), "f"(used.bc0.x), "f"(used.bc0.y),
                     "f"(used.bc1.x), "f"(used.bc1.y), "f"(used.de.x), "f"(used.de.y));
#pragma unroll
        for (int k = 0; k < 10; ++k) nm[k] = __ldg(p + 64 * (5 + PPB_PERM[DIR][k]));
    }
    template <int S> __device__ __forceinline__ void store(int i, const float (&h)[5], const float (&m)[10], bool = true) {
        float* __restrict__ p = pout + off(i);
        p[0] = h[0];
        p[64 * Dir<DIR>::U] = h[1];
        p[64 * Dir<DIR>::V] = h[2];
        p[64 * Dir<DIR>::W] = h[3];
        p[64 * 4] = h[4];
#pragma unroll
        for (int k = 0; k < 10; ++k) p[64 * (5 + PPB_PERM[DIR][k])] = m[k];
    }
    // PPB-only sweep: the hydro fields of the cell are copied through unchanged
    template <int S> __device__ __forceinline__ void store_ppb(int i, const float (&m)[10]) {
        const long long o = off(i);
        float* __restrict__ p = pout + o;
        const float* __restrict__ q = pin + o;
#pragma unroll
        for (int f = 0; f < 5; ++f) p[64 * f] = __ldg(q + 64 * f);
#pragma unroll
        for (int k = 0; k < 10; ++k) p[64 * (5 + PPB_PERM[DIR][k])] = m[k];
    }
    __device__ __forceinline__ void finish() {}
};

// thread -> pencil: 16 lanes = the 4x4 transverse cells of one brick column; a CTA of 128 threads = 8 brick
// columns adjacent along a.  (a, b) = the two transverse axes in increasing axis order.
template <int DIR, int GRAV, bool FLAT, bool TWOF>
__global__ void __maxnreg__(PPM_MAXREG) ppm_sweep_kernel(const SweepParams P) {
    constexpr int AXA = (DIR == 0) ? 1 : 0, AXB = (DIR == 2) ? 1 : 2;
    const int t = threadIdx.x;
    const int ba = blockIdx.x * (PPM_CTA / 16) + (t >> 4), bb = blockIdx.y;
    const int a = ba * 4 + (t & 3), b = bb * 4 + ((t >> 2) & 3);
    // the lanes that march: taken by a full-warp vote BEFORE the pad lanes leave (__activemask() after a divergent
    // return need not equal the set of lanes that stay)
    const unsigned wmask = __ballot_sync(0xffffffffu, a < P.na && b < P.nb);
    if (a >= P.na || b >= P.nb) return;
    const int c0 = blockIdx.z * P.chunk;
    const int c1 = min(c0 + P.chunk, P.n);
    const long long tb = (long long)ba * P.SBa + (long long)bb * P.SBb + (((t & 3) << (2 * AXA)) + (((t >> 2) & 3) << (2 * AXB)));
    IoDirect<DIR> io(P, tb, c0 - PPM_NGHOST, c0);
    const float* pflat = FLAT ? P.flat + ((long long)ba * P.FBa + (long long)bb * P.FBb + (((t & 3) << (2 * AXA)) + (((t >> 2) & 3) << (2 * AXB)))) : nullptr;
    float vmax = 0.f;
    march<DIR, GRAV, FLAT, false, false, TWOF>(P, io, a, b, c0, c1, true, wmask, pflat, vmax, Segment(), nullptr, TWOF ? P.in + tb + 5 * 64 : nullptr);
}

// PPB-only sweep (NEXT-2), direct path
template <int DIR>
__global__ void __launch_bounds__(PPM_CTA) ppm_advect_kernel(const SweepParams P) {
    constexpr int AXA = (DIR == 0) ? 1 : 0, AXB = (DIR == 2) ? 1 : 2;
    const int t = threadIdx.x;
    const int ba = blockIdx.x * (PPM_CTA / 16) + (t >> 4), bb = blockIdx.y;
    const int a = ba * 4 + (t & 3), b = bb * 4 + ((t >> 2) & 3);
    if (a >= P.na || b >= P.nb) return;
    const int c0 = blockIdx.z * P.chunk;
    const int c1 = min(c0 + P.chunk, P.n);
    const long long tb = (long long)ba * P.SBa + (long long)bb * P.SBb + (((t & 3) << (2 * AXA)) + (((t >> 2) & 3) << (2 * AXB)));
    IoDirect<DIR> io(P, tb, c0 - PPM_NGHOST, c0);
    march_ppb<DIR>(P, io, c0, c1);
}

// ---- shared-memory / mbarrier / bulk-copy primitives ----------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    // Called by whole warps.  The loop exit is a warp vote, i.e. provably uniform: a per-lane spin loop (in C++ or
    // hidden inside the asm) makes ptxas treat everything after it as divergent and give up the uniform datapath
    // for the marching loop's index arithmetic.
    const uint32_t addr = smem_u32(bar);
    uint32_t done;
    do {
        asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}\n"
                     : "=r"(done) : "r"(addr), "r"(parity) : "memory");
    } while (!__all_sync(0xffffffffu, done));   // warp-uniform exit: every lane polls, the vote decides
}
__device__ __forceinline__ void tma_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void tma_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void tma_wait_all0() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// =====================================================================================================
// IoBulk: every sweep direction (sweep-axis extent a multiple of 4).  Warp = 2 brick columns adjacent along a.
// A brick record keeps its 15 fields contiguous, so the hydro part (5 fields, 1280 B) and the PPB part (10
// fields, 2560 B) of a brick are plain 1-D bulk copies (cp.async.bulk, no tensor map): global -> shared when the
// brick comes up, shared -> global when its four cells are finished.  Nothing else touches global memory, so
// DRAM sees whole 1280/2560-byte runs in all three directions, no load sits in a register waiting, and the
// marching body needs no prefetch registers.
//
// Results are written IN PLACE over the brick's own input in shared memory: cell i's hydro input is read at
// iteration n = i and its PPB input at n = i + 3, its results are written at n = i + 4.  So a hydro slot lives
// for 3 bricks of marching (input, output, in flight to global) and a PPB slot for 2: rings of 3 and 2 slots,
// 17.8 KB per warp, 12 warps per SM.
// =====================================================================================================
// ADV: the split PPB-only sweeps stage one hydro field per brick, so the hydro slots shrink and four CTAs fit an SM
template <int DIR, bool ADV = false> struct BulkGeom {
    static constexpr int AXA = (DIR == 0) ? 1 : 0, AXB = (DIR == 2) ? 1 : 2;
    // the second brick of a slot is shifted so that the two half warps fall on different banks where the
    // direction allows it (z: 16 lanes contiguous; y: 4-float runs 16 apart; x: every 4th bank, 4-way inherent)
    static constexpr int PAD = (DIR == 2) ? 16 : ((DIR == 1) ? 8 : 4);
    static constexpr int HB = 5 * 64, PB = 10 * 64;             // floats per brick record: hydro part, PPB part
    static constexpr int HBS = ADV ? 64 : HB;                   // floats of a brick's hydro part in shared memory
    static constexpr int HSLOT = 2 * HBS + PAD, PSLOT = 2 * PB + PAD;
    static constexpr int NH = 3, NP = 2;                        // ring depths
    static constexpr int WARP_FLOATS = NH * HSLOT + NP * PSLOT;
    static constexpr int WARPS = PPM_BULK_WARPS;                // warps per CTA (build knob; 12 warps are resident per SM)
    static constexpr int CTAS = (ADV ? 16 : 12) / PPM_BULK_WARPS;   // resident CTAs per SM the launch bounds ask for
    static constexpr size_t SMEM = (size_t)WARPS * WARP_FLOATS * 4 + WARPS * (NH + NP) * sizeof(uint64_t);
};

__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void bulk_s2g(void* dst, const void* src, uint32_t bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(smem_u32(src)), "r"(bytes) : "memory");
}

// The same operations predicated on `lead` inside the asm (lead = lane 0).  The statement is executed by the whole, converged
// warp with warp-uniform operands, so ptxas issues the bulk copy once under a predicate instead of wrapping it, inside an
// `if (lane == 0)` region, into a lane-election loop of its own (five more instructions per copy).
__device__ __forceinline__ void mbar_expect_tx_p(bool lead, uint64_t* bar, uint32_t bytes) {
    asm volatile("{\n.reg .pred q;\n.reg .pred e;\nelect.sync _|e, 0xffffffff;\nsetp.ne.b32 q, %2, 0;\nand.pred q, q, e;\n@q mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n}\n"
                 ::"r"(smem_u32(bar)), "r"(bytes), "r"((int)lead) : "memory");
}
__device__ __forceinline__ void bulk_g2s_p(bool lead, void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("{\n.reg .pred q;\n.reg .pred e;\nelect.sync _|e, 0xffffffff;\nsetp.ne.b32 q, %4, 0;\nand.pred q, q, e;\n@q cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n}\n"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)), "r"((int)lead) : "memory");
}
__device__ __forceinline__ void bulk_s2g_p(bool lead, void* dst, const void* src, uint32_t bytes) {
    asm volatile("{\n.reg .pred q;\n.reg .pred e;\nelect.sync _|e, 0xffffffff;\nsetp.ne.b32 q, %3, 0;\nand.pred q, q, e;\n@q cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;\n}\n"
                 ::"l"(dst), "r"(smem_u32(src)), "r"(bytes), "r"((int)lead) : "memory");
}
__device__ __forceinline__ void tma_commit_p(bool lead) {
    asm volatile("{\n.reg .pred q;\n.reg .pred e;\nelect.sync _|e, 0xffffffff;\nsetp.ne.b32 q, %0, 0;\nand.pred q, q, e;\n@q cp.async.bulk.commit_group;\n}\n" ::"r"((int)lead) : "memory");
}
__device__ __forceinline__ void tma_wait_read0_p(bool lead) {
    asm volatile("{\n.reg .pred q;\n.reg .pred e;\nelect.sync _|e, 0xffffffff;\nsetp.ne.b32 q, %0, 0;\nand.pred q, q, e;\n@q cp.async.bulk.wait_group.read 0;\n}\n" ::"r"((int)lead) : "memory");
}

// ADV: the PPB-only sweeps (NEXT-2) — of a brick's hydro part only the velocity component along the sweep axis is staged (one
// 256-byte field, from the buffer that holds the hydro fields: P.in + P.hdelta) and only its PPB part goes back to global memory.
template <int DIR, bool ADV = false>
struct IoBulk {
    using G = BulkGeom<DIR, ADV>;
    static constexpr int HOFF = ADV ? 64 * Dir<DIR>::U : 0;          // first float of a record's hydro part that is staged
    static constexpr int HBYTES = G::HBS * 4;                       // bytes of it
    static constexpr int FU = ADV ? 0 : 64 * Dir<DIR>::U;            // where the normal velocity sits in a staged hydro part
    static constexpr int SH = 2 * DIR;   // in-brick stride along the sweep axis = 1 << SH floats
    const SweepParams& P;
    float* const hyd;            // warp's hydro ring [NH][HSLOT], already offset to the lane's layer-0 element
    float* const ppr;            // warp's PPB ring   [NP][PSLOT], same
    float* const hyd0;           // ring bases as the bulk copies see them (lane 0 uses them)
    float* const ppr0;
    uint64_t* const bar;         // [0..NH) hydro slots, [NH..NH+NP) PPB slots
    const int lane;
    const long long gcol;        // float offset of the warp's first brick column (brick 0 along the sweep axis)
    const long long hcol;        // the same column inside a halo layer (PPM_BC_HALO: one brick layer of a neighbouring sub-domain)
    const int ncol;              // brick columns of this warp that exist (1 or 2)
    const int k0, kend;          // first / last brick index along the sweep axis this pencil segment touches (ghosts included)
    // per-brick state, refreshed when a new brick comes up (once per 4 iterations); everything is warp-uniform
    int hs, ps;                  // ring slot of the hydro brick being read / of the PPB brick being read
    unsigned ph;                 // bit j: phase the next wait on mbarrier j (0..NH-1 hydro slots, NH.. PPB slots) must see; lives across pencil segments
    int hcur, hprv;              // float offset (from hyd) of the hydro slot being read / of the one receiving results
    int pcur, pst;               // float offset (from ppr) of the PPB slot being read / of the one receiving results
    int hrev, prev;              // 3 if the brick being read is a mirror image (cells taken in reverse, odd fields negated), else 0
    int jb;                      // image index of the hydro brick's cell 0

    __device__ __forceinline__ IoBulk(const SweepParams& P_, float* wsm, uint64_t* wbar, unsigned ph_, int lane_, long long gcol_, int ncol_, int c0, int c1,
                                      long long hcol_ = 0)
        : P(P_),
          hyd(wsm + (lane_ >> 4) * (G::HBS + G::PAD) + ((lane_ & 3) << (2 * G::AXA)) + (((lane_ >> 2) & 3) << (2 * G::AXB))),
          ppr(wsm + G::NH * G::HSLOT + (lane_ >> 4) * (G::PB + G::PAD) + ((lane_ & 3) << (2 * G::AXA)) + (((lane_ >> 2) & 3) << (2 * G::AXB))),
          hyd0(wsm), ppr0(wsm + G::NH * G::HSLOT), bar(wbar), lane(lane_), gcol(gcol_), hcol(hcol_), ncol(ncol_), k0(c0 / 4 - 1), kend(c1 / 4),
          ph(ph_), hs(0), ps(0), hcur(0), hprv(0), pcur(0), pst(0), hrev(0), prev(0), jb(0) {
        if (lane == 0) {
#pragma unroll
            for (int j = 0; j < G::NH; ++j) if (k0 + j <= kend) issue_hydro(k0 + j, j);
#pragma unroll
            for (int j = 0; j < G::NP; ++j) if (k0 + j <= kend) issue_ppb(k0 + j, j);
        }
    }
    // brick holding chunk k (ghost chunks map onto their periodic / mirror image; mirrored ones are read reversed)
    __device__ __forceinline__ int chunk_brick(int k, int& rev) const {
        rev = 0;
        const int nk = P.nbrick_d;
        if ((unsigned)k < (unsigned)nk) return k;
        if (k < 0) { if (P.bc_lo == PPM_BC_HALO) return k; if (P.bc_lo == PPM_BC_PERIODIC) return nk - 1; rev = 3; return 0; }
        if (P.bc_hi == PPM_BC_HALO) return k;                  // (a halo brick keeps its own index: its cells sit where they are)
        if (P.bc_hi == PPM_BC_PERIODIC) return 0;
        rev = 3; return nk - 1;
    }
    // record of chunk k in the warp's first brick column, and the stride to its second column: the state buffer, or — for the
    // one ghost chunk beyond a PPM_BC_HALO face — the halo layer received from the neighbouring sub-domain
    __device__ __forceinline__ const float* brick_src(int k, long long& stride2) const {
        if (k < 0 && P.bc_lo == PPM_BC_HALO) { stride2 = P.HBa; return P.halo_lo + hcol; }
        if (k >= P.nbrick_d && P.bc_hi == PPM_BC_HALO) { stride2 = P.HBa; return P.halo_hi + hcol; }
        int rev; const int bd = chunk_brick(k, rev);
        stride2 = P.SBa;
        return P.in + gcol + (long long)bd * P.SBd;
    }
    // steady state, whole warp: the same two issues with the leader predicate inside the asm
    __device__ __forceinline__ void issue_hydro_w(bool lead, const float* src, long long st2, int slot) {
        mbar_expect_tx_p(lead, bar + slot, ncol * G::HB * 4);
        bulk_g2s_p(lead, hyd0 + slot * G::HSLOT, src, G::HB * 4, bar + slot);
        bulk_g2s_p(lead && ncol > 1, hyd0 + slot * G::HSLOT + G::HBS + G::PAD, src + st2, G::HB * 4, bar + slot);
    }
    __device__ __forceinline__ void issue_ppb_w(bool lead, const float* src, long long st2, int slot) {
        mbar_expect_tx_p(lead, bar + G::NH + slot, ncol * G::PB * 4);
        bulk_g2s_p(lead, ppr0 + slot * G::PSLOT, src + G::HB, G::PB * 4, bar + G::NH + slot);
        bulk_g2s_p(lead && ncol > 1, ppr0 + slot * G::PSLOT + G::PB + G::PAD, src + G::HB + st2, G::PB * 4, bar + G::NH + slot);
    }
    // src = the record of the wanted brick in the warp's first column, st2 = stride to its second column
    __device__ __forceinline__ void issue_hydro_at(const float* src, long long st2, int slot) {       // lane 0 only
        if (ADV) src += P.hdelta + HOFF;
        mbar_expect_tx(bar + slot, ncol * HBYTES);
        bulk_g2s(hyd0 + slot * G::HSLOT, src, HBYTES, bar + slot);
        if (ncol > 1) bulk_g2s(hyd0 + slot * G::HSLOT + G::HBS + G::PAD, src + st2, HBYTES, bar + slot);
    }
    __device__ __forceinline__ void issue_ppb_at(const float* src, long long st2, int slot) {         // lane 0 only
        mbar_expect_tx(bar + G::NH + slot, ncol * G::PB * 4);
        bulk_g2s(ppr0 + slot * G::PSLOT, src + G::HB, G::PB * 4, bar + G::NH + slot);
        if (ncol > 1) bulk_g2s(ppr0 + slot * G::PSLOT + G::PB + G::PAD, src + G::HB + st2, G::PB * 4, bar + G::NH + slot);
    }
    __device__ __forceinline__ void issue_hydro(int k, int slot) { long long st2; const float* src = brick_src(k, st2); issue_hydro_at(src, st2, slot); }
    __device__ __forceinline__ void issue_ppb(int k, int slot) { long long st2; const float* src = brick_src(k, st2); issue_ppb_at(src, st2, slot); }
    __device__ __forceinline__ void wait_slot(int j) {        // whole warp
        mbar_wait(bar + j, (ph >> j) & 1);
        ph ^= 1u << j;
    }
    // S = -1: run-time brick phase, ghost bricks and segment ends handled.  S = 0..3: steady state — n & 3 == S, the
    // bricks in play are interior bricks that are neither the first nor the last of the segment (march()).
    template <int S> __device__ __forceinline__ void begin(int n) {
        const int s = (S >= 0 && S < 4) ? S : (n & 3);
        if (s == 0) {                                          // a new hydro brick k comes up; results of brick k - 1 start
            const int k = n >> 2;
            pst = pcur;                                        // PPB brick k - 1 is the one being read since n - 1
            hprv = hcur;
            if (S >= 0 || k != k0) {
                hs = (hs == G::NH - 1) ? 0 : hs + 1;
                hcur = hs * G::HSLOT;
            } else {
                chunk_brick(k0, prev);                         // the very first PPB cell (c0 - 1) is the last cell of brick k0
                wait_slot(G::NH);
            }
            if (S >= 0) { jb = n; hrev = 0; }
            else jb = chunk_brick(k, hrev) * 4;
            wait_slot(hs);
        } else if (s == 1) {
            // ring refill, once per brick, one full iteration after brick k - 2 was shipped (so its bulk stores have
            // long read their slots and lane 0 does not wait here).  Hydro brick k sits in slot hs and brick k - 1
            // (receiving results) in hs - 1, so the dead hydro slot is hs + 1 (mod 3); the PPB brick being read is
            // k - 1 in slot ps, the dead one is ps ^ 1.
            const int k = n >> 2;
            if (S >= 0 || k != k0) {
                __syncwarp();
#ifdef PPM_DEBUG_POISON
                // debug build (compute-sanitizer's racecheck is not available on this pool): once the bulk stores that read
                // the two dead slots have completed, every lane fills them with NaN before the refill is issued.  A lane
                // that reads a slot before its load has landed, or a slot other than the one it should, then produces NaN
                // instead of plausible stale data, and the parity tests fail loudly.
                if (lane == 0) tma_wait_read0();
                __syncwarp();
                {
                    const int dh = (hs == G::NH - 1 ? 0 : hs + 1) * G::HSLOT, dp = (ps ^ 1) * G::PSLOT;
                    const bool rh = S >= 0 || (k + 1 >= k0 + G::NH && k + 1 <= kend), rp = S >= 0 || (k >= k0 + G::NP && k <= kend);
                    for (int e = lane; e < G::HSLOT; e += 32) if (rh) hyd0[dh + e] = __int_as_float(0x7fc00000);
                    for (int e = lane; e < G::PSLOT; e += 32) if (rp) ppr0[dp + e] = __int_as_float(0x7fc00000);
                    fence_async_smem();
                    __syncwarp();
                }
#endif
                if (S >= 0 && PPM_PRED_COPIES) {
                    // steady state: brick k is an interior brick of the state buffer — no image, no halo layer; only brick
                    // k + 1 can be the ghost brick beyond the high end (its record comes from brick_src then)
                    const bool lead = true;            // (the leader is elected inside the asm; `lead` carries the warp-uniform condition)
                    tma_wait_read0_p(lead);
                    const float* rec = P.in + gcol + (long long)k * P.SBd;
                    long long st2 = P.SBa;
                    const float* nxt = rec + P.SBd;
                    if (k + 1 >= P.nbrick_d) nxt = brick_src(k + 1, st2);
                    issue_hydro_w(lead, nxt, st2, hs == G::NH - 1 ? 0 : hs + 1);
                    issue_ppb_w(lead, rec, P.SBa, ps ^ 1);
                } else if (lane == 0) {
                    tma_wait_read0();
                    if (S >= 0) {
                        const float* rec = P.in + gcol + (long long)k * P.SBd;
                        if (k + 1 < P.nbrick_d) issue_hydro_at(rec + P.SBd, P.SBa, hs == G::NH - 1 ? 0 : hs + 1);
                        else issue_hydro(k + 1, hs == G::NH - 1 ? 0 : hs + 1);
                        issue_ppb_at(rec, P.SBa, ps ^ 1);
                    } else {
                        if (k + 1 >= k0 + G::NH && k + 1 <= kend) issue_hydro(k + 1, hs == G::NH - 1 ? 0 : hs + 1);
                        if (k >= k0 + G::NP && k <= kend) issue_ppb(k, ps ^ 1);
                    }
                }
            }
        } else if (s == 3) {                                   // PPB cell c = n - 3 is the first of brick c >> 2
            const int k = (n - 3) >> 2;
            if (S >= 0 || k > k0) {
                ps ^= 1;
                pcur = ps * G::PSLOT;
                if (S >= 0) prev = 0; else chunk_brick(k, prev);
                wait_slot(G::NH + ps);
            }
        }
    }
    template <int S> __device__ __forceinline__ void hydro(int n, int& j, float& sgn, float (&v)[5]) {
        if (S >= 0) {                                          // interior brick, cells in order
            sgn = 1.0f;
            j = n;
            const float* src = hyd + hcur + (((S < 4) ? S : (n & 3)) << SH);
            v[0] = src[0];
            v[1] = src[FU];
            v[2] = src[64 * Dir<DIR>::V];
            v[3] = src[64 * Dir<DIR>::W];
            v[4] = src[64 * 4];
            return;
        }
        const int s = (n & 3) ^ hrev;
        sgn = hrev ? -1.0f : 1.0f;
        j = jb + s;
        const float* src = hyd + hcur + (s << SH);
        const float un = src[FU];
        v[1] = hrev ? -un : un;                                // normal velocity: odd under the mirror
        if (ADV) { v[0] = v[2] = v[3] = v[4] = 0.f; return; }   // (the PPB-only sweeps stage nothing else)
        v[0] = src[0];
        v[2] = src[64 * Dir<DIR>::V];
        v[3] = src[64 * Dir<DIR>::W];
        v[4] = src[64 * 4];
    }
    template <int S> __device__ __forceinline__ void ppb(int c, float (&m)[10]) {
        const int s = (S >= 0 && S < 4) ? ((S + 1) & 3) : ((S >= 4) ? (c & 3) : ((c & 3) ^ prev));      // c = n - 3
        const float* src = ppr + pcur + (s << SH);
#pragma unroll
        for (int q = 0; q < 10; ++q) m[q] = src[64 * PPB_PERM[DIR][q]];
        if (S < 0 && prev) { m[1] = -m[1]; m[4] = -m[4]; m[6] = -m[6]; }   // odd coefficients under the mirror (warp-uniform, rare)
    }
    __device__ __forceinline__ void ppb_prefetch(int, const PpbCell&) {}
    static constexpr bool HAS_OLD = true;
    static constexpr bool HAS_FAST = true;
    // the hydro input of interior cell i, still in its slot when the cell is finished (n = i + 4)
    template <int S> __device__ __forceinline__ void old_hydro(int i, float (&v)[5]) {
        const float* src = hyd + hprv + (((S >= 0 && S < 4) ? S : (i & 3)) << SH);
        v[0] = src[0];
        v[1] = src[64 * Dir<DIR>::U];
        v[2] = src[64 * Dir<DIR>::V];
        v[3] = src[64 * Dir<DIR>::W];
        v[4] = src[64 * 4];
    }
    // finished cell i, written over its own input (already consumed: hydro at n = i, PPB at n = i + 3 < i + 4)
    // (keep = false: a solid cell of the confining sphere — its slot entries stay what they are, the input)
    template <int S> __device__ __forceinline__ void store(int i, const float (&h)[5], const float (&m)[10], bool keep = true) {
        const int s = (S >= 0 && S < 4) ? S : (i & 3);         // i = n - 4
        float* dh = hyd + hprv + (s << SH);
        if (keep) {
            dh[0] = h[0];
            dh[64 * Dir<DIR>::U] = h[1];
            dh[64 * Dir<DIR>::V] = h[2];
            dh[64 * Dir<DIR>::W] = h[3];
            dh[64 * 4] = h[4];
        }
        store_ppb<S>(i, m, keep);
    }
    // PPB part of cell i only (PPB-only sweep: the hydro slot goes back to global memory as it came in)
    template <int S> __device__ __forceinline__ void store_ppb(int i, const float (&m)[10], bool keep = true) {
        const int s = (S >= 0 && S < 4) ? S : (i & 3);
        float* dp = ppr + pst + (s << SH);
        if (keep) {
#pragma unroll
            for (int q = 0; q < 10; ++q) dp[64 * PPB_PERM[DIR][q]] = m[q];
        }
        if (s == 3) {                                          // brick i >> 2 is complete: ship it
            fence_async_smem();                                // generic-proxy writes -> visible to the async proxy
            __syncwarp();
            if (S >= 0 && PPM_PRED_COPIES) {
                const bool lead = true;
                float* dst = P.out + gcol + (long long)(i >> 2) * P.SBd;
                const float* sh = hyd0 + hprv;
                const float* sp = ppr0 + pst;
                bulk_s2g_p(lead, dst, sh, G::HB * 4);
                bulk_s2g_p(lead, dst + G::HB, sp, G::PB * 4);
                bulk_s2g_p(lead && ncol > 1, dst + P.SBa, sh + G::HBS + G::PAD, G::HB * 4);
                bulk_s2g_p(lead && ncol > 1, dst + P.SBa + G::HB, sp + G::PB + G::PAD, G::PB * 4);
                tma_commit_p(lead);
            } else if (lane == 0) {
                float* dst = P.out + gcol + (long long)(i >> 2) * P.SBd;
                const float* sh = hyd0 + hprv;
                const float* sp = ppr0 + pst;
                if (!ADV) bulk_s2g(dst, sh, G::HB * 4);
                bulk_s2g(dst + G::HB, sp, G::PB * 4);
                if (ncol > 1) {
                    if (!ADV) bulk_s2g(dst + P.SBa, sh + G::HBS + G::PAD, G::HB * 4);
                    bulk_s2g(dst + P.SBa + G::HB, sp + G::PB + G::PAD, G::PB * 4);
                }
                tma_commit();
            }
        }
    }
    __device__ __forceinline__ void finish() {
        if (lane == 0) tma_wait_all0();                        // smem must outlive the last bulk store
        __syncwarp();
    }
};

// One CTA = one segment of one pencil tile (8 x 1 brick columns).  Tiles [0, P.tiles_a) are cut into segments of
// P.chunk cells, the remaining tiles into segments of P.chunk_b cells (both multiples of 4): the launcher marches
// whole pencils while they fill complete waves of resident CTAs and cuts the pencils of the ragged last wave into
// shorter segments, so that the SMs run dry together.  A cut costs 8 redundant warm-up cells; results do not
// depend on where the cuts are.
// this CTA's pencil segment: tile index and cell range [c0, c1)
__device__ __forceinline__ void bulk_segment(const SweepParams& P, int& tile, int& c0, int& c1) {
    const int ncha = (P.n + P.chunk - 1) / P.chunk;
    const int na_ctas = P.tiles_a * ncha;
    int u = blockIdx.x, ch = P.chunk, nch = ncha, t0 = 0;
    if (u >= na_ctas) { u -= na_ctas; ch = P.chunk_b; nch = (P.n + ch - 1) / ch; t0 = P.tiles_a; }
    const int t = u / nch;
    tile = t0 + t;
    c0 = (u - t * nch) * ch;
    c1 = min(c0 + ch, P.n);
}
template <int DIR>
__device__ __forceinline__ void bulk_init_barriers(uint64_t* bars) {
    using G = BulkGeom<DIR>;
    if (threadIdx.x < G::WARPS * (G::NH + G::NP)) mbar_init(bars + threadIdx.x, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    fence_async_smem();
    __syncthreads();
}

// Confining sphere: a warp none of whose pencils holds a fluid cell (48 % of the pencils of a cube lie wholly outside its
// inscribed sphere) only has to pass its brick records on to the other buffer: whole-record bulk copies through two
// slots of the warp's ring memory, no arithmetic.
template <int DIR>
__device__ __forceinline__ unsigned bulk_copy_through(const SweepParams& P, float* wsm, uint64_t* bar, int lane, long long gcol, int ncol, int c0, int c1,
                                                      unsigned ph) {      // ph: mbarrier phases (bits 0, 1 are used), handed on to the caller
    constexpr int REC = PPM_BRICK_FLOATS;                      // floats per brick record
    const int kb = c0 >> 2, ke = c1 >> 2;
    if (kb >= ke) return ph;
    if (lane == 0) {
#pragma unroll 1
        for (int j = 0; j < 2 && kb + j < ke; ++j) {
            const float* src = P.in + gcol + (long long)(kb + j) * P.SBd;
            mbar_expect_tx(bar + j, ncol * REC * 4);
            bulk_g2s(wsm + j * 2 * REC, src, REC * 4, bar + j);
            if (ncol > 1) bulk_g2s(wsm + j * 2 * REC + REC, src + P.SBa, REC * 4, bar + j);
        }
    }
#pragma unroll 1
    for (int k = kb; k < ke; ++k) {
        const int j = (k - kb) & 1;
        mbar_wait(bar + j, (ph >> j) & 1);
        ph ^= 1u << j;
        if (lane == 0) {
            float* dst = P.out + gcol + (long long)k * P.SBd;
            bulk_s2g(dst, wsm + j * 2 * REC, REC * 4);
            if (ncol > 1) bulk_s2g(dst + P.SBa, wsm + j * 2 * REC + REC, REC * 4);
            tma_commit();
            if (k + 2 < ke) {
                tma_wait_read0();                              // the store just issued has read the slot: refill it
                const float* src = P.in + gcol + (long long)(k + 2) * P.SBd;
                mbar_expect_tx(bar + j, ncol * REC * 4);
                bulk_g2s(wsm + j * 2 * REC, src, REC * 4, bar + j);
                if (ncol > 1) bulk_g2s(wsm + j * 2 * REC + REC, src + P.SBa, REC * 4, bar + j);
            }
        }
        __syncwarp();
    }
    if (lane == 0) tma_wait_all0();
    __syncwarp();
    return ph;
}

template <int DIR, int GRAV, bool FLAT, bool CFL, bool SPH, bool TWOF>
__global__ void __launch_bounds__(BulkGeom<DIR>::WARPS * 32, BulkGeom<DIR>::CTAS) ppm_sweep_bulk_kernel(const SweepParams P) {
    using G = BulkGeom<DIR>;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float* sm = reinterpret_cast<float*>(smem_raw);
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem_raw + (size_t)G::WARPS * G::WARP_FLOATS * 4);
    // (the shuffle tells the compiler that the warp index is warp-uniform: ring addresses, mbarriers and the bulk-copy
    // operands then live in uniform registers and the copies are issued without a lane-election loop)
    const int warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0), lane = threadIdx.x & 31;
    bulk_init_barriers<DIR>(bars);
    const int nba = (P.na + 3) >> 2;
    const int ntx = (nba + 2 * G::WARPS - 1) / (2 * G::WARPS);    // tiles along a
    int tile, c0, c1;
    bulk_segment(P, tile, c0, c1);
    const int bb = tile / ntx, tx = tile - bb * ntx;
    const int ba0 = (tx * G::WARPS + warp) * 2;                    // the warp's brick columns: ba0, ba0 + 1 along a; bb along b
    if (ba0 >= nba) return;                                        // whole warp out of range (no block-wide sync below)
    const int a = (ba0 + (lane >> 4)) * 4 + (lane & 3);
    const int b = bb * 4 + ((lane >> 2) & 3);
    const long long gcol = (long long)ba0 * P.SBa + (long long)bb * P.SBb;
    Segment seg;
    unsigned ph0 = 0;
    const int c0s = c0, c1s = c1;                                  // this CTA's pencil segment
    if (SPH) {
        // The warp marches only the bricks that hold fluid cells of its 32 pencils; the bricks before and after pass through
        // untouched (the ghost cells beyond a lane's segment are mirror images read per lane, never these bricks).
        seg = sphere_segment<DIR>(P, a, b);
        const bool has = a < P.na && b < P.nb && seg.lo <= seg.hi;
        const int lo_w = __reduce_min_sync(0xffffffffu, has ? seg.lo : 0x7fffffff), hi_w = __reduce_max_sync(0xffffffffu, has ? seg.hi : -1);
        const int c0w = max(c0, lo_w & ~3), c1w = min(c1, (hi_w + 4) & ~3);
        float* wsm = sm + warp * G::WARP_FLOATS;
        uint64_t* wbar = bars + warp * (G::NH + G::NP);
        if (hi_w < 0 || c0w >= c1w) {                               // nothing but solid cells under this warp in this segment
            bulk_copy_through<DIR>(P, wsm, wbar, lane, gcol, min(2, nba - ba0), c0, c1, 0u);
            return;
        }
        ph0 = bulk_copy_through<DIR>(P, wsm, wbar, lane, gcol, min(2, nba - ba0), c0, c0w, 0u);
        c0 = c0w; c1 = c1w;
    }
    IoBulk<DIR> io(P, sm + warp * G::WARP_FLOATS, bars + warp * (G::NH + G::NP), ph0, lane, gcol, min(2, nba - ba0), c0, c1,
                   (long long)ba0 * P.HBa + (long long)bb * P.HBb);
    if (PPM_PRED_COPIES) {
        // The steady-state body issues its bulk copies from the lane elect.sync picks, the generic body from lane 0, and bulk
        // async-groups belong to the thread that committed them: the two must be the same lane (they are: the lowest one).
        // Checked once per warp; a mismatch raises the state flag (PPM_ESTATE) instead of racing silently.
        unsigned e;
        asm volatile("{\n.reg .pred q;\nelect.sync _|q, 0xffffffff;\nselp.u32 %0, 1, 0, q;\n}\n" : "=r"(e));
        if ((e != 0) != (lane == 0)) atomicOr(P.flag, 2);
    }
    // pad pencils of a ragged grid (and the lanes of a missing second brick column) compute garbage that is never read
    const float* pflat = FLAT ? P.flat + ((long long)min(ba0 + (lane >> 4), nba - 1) * P.FBa + (long long)bb * P.FBb +
                                          (((lane & 3) << (2 * G::AXA)) + (((lane >> 2) & 3) << (2 * G::AXB)))) : nullptr;
    const bool valid = a < P.na && b < P.nb;
    float vmax = 0.f;
    if (SPH) {
        const float* gpen = P.in + gcol + (long long)(lane >> 4) * P.SBa + (((lane & 3) << (2 * G::AXA)) + (((lane >> 2) & 3) << (2 * G::AXB)));
        march<DIR, GRAV, FLAT, CFL, true, false>(P, io, a, b, c0, c1, valid, 0xffffffffu, pflat, vmax, seg, gpen);
        bulk_copy_through<DIR>(P, sm + warp * G::WARP_FLOATS, bars + warp * (G::NH + G::NP), lane, gcol, min(2, nba - ba0), c1, c1s, io.ph);
        (void)c0s;
    } else {
        // two-fluid EOS: the lane's pencil of m000 in the input buffer (pad lanes of a ragged grid read their clamped column)
        const float* mpen = TWOF ? P.in + ((long long)min(ba0 + (lane >> 4), nba - 1) * P.SBa + (long long)bb * P.SBb + 5 * 64 +
                                           (((lane & 3) << (2 * G::AXA)) + (((lane >> 2) & 3) << (2 * G::AXB)))) : nullptr;
        march<DIR, GRAV, FLAT, CFL, false, TWOF>(P, io, a, b, c0, c1, valid, 0xffffffffu, pflat, vmax, Segment(), nullptr, mpen);
    }
    if (CFL) {
        // warp max by one REDUX on the bit patterns (non-negative floats order like unsigned integers; a NaN has the
        // largest pattern and so survives: ppm_cfl_dt reports it), then one atomicMax per warp
        const unsigned m = __reduce_max_sync(0xffffffffu, valid ? __float_as_uint(fmaxf(vmax, 0.f)) : 0u);
        if (lane == 0) atomicMax(P.cflmax, m);
    }
}

// PPB-only sweep (NEXT-2), bulk-staged path: same rings; the hydro fields stay where they are (the buffer P.in + P.hdelta) and
// only the PPB part of every brick is written to P.out — the launcher keeps track of which buffer holds which part
// (SPLIT = false: whole records in, whole records out — grids on which another axis takes the direct path)
template <int DIR, bool SPLIT>
__global__ void __launch_bounds__(BulkGeom<DIR, SPLIT>::WARPS * 32, BulkGeom<DIR, SPLIT>::CTAS) ppm_advect_bulk_kernel(const SweepParams P) {
    using G = BulkGeom<DIR, SPLIT>;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float* sm = reinterpret_cast<float*>(smem_raw);
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem_raw + (size_t)G::WARPS * G::WARP_FLOATS * 4);
    // (the shuffle tells the compiler that the warp index is warp-uniform: ring addresses, mbarriers and the bulk-copy
    // operands then live in uniform registers and the copies are issued without a lane-election loop)
    const int warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0), lane = threadIdx.x & 31;
    bulk_init_barriers<DIR>(bars);
    const int nba = (P.na + 3) >> 2;
    const int ntx = (nba + 2 * G::WARPS - 1) / (2 * G::WARPS);
    int tile, c0, c1;
    bulk_segment(P, tile, c0, c1);
    const int bb = tile / ntx, tx = tile - bb * ntx;
    const int ba0 = (tx * G::WARPS + warp) * 2;
    if (ba0 >= nba) return;
    const long long gcol = (long long)ba0 * P.SBa + (long long)bb * P.SBb;
    IoBulk<DIR, SPLIT> io(P, sm + warp * G::WARP_FLOATS, bars + warp * (G::NH + G::NP), 0u, lane, gcol, min(2, nba - ba0), c0, c1);
    march_ppb<DIR>(P, io, c0, c1);
}

// cells per segment for the tiles of the ragged last wave: the cut that minimises (waves of segments) x (segment
// length + 8 warm-up cells); ntail tiles, slots resident CTAs, n cells per pencil
int ppm_tail_chunk_impl(int ntail, int slots, int n) {
    int best = n;
    double best_t = 1e300;
    for (int np = 1; np <= 8; ++np) {
        const int ch = ((n + np - 1) / np + 3) / 4 * 4;
        if (ch < 32 && np > 1) break;
        const int nch = (n + ch - 1) / ch;
        const long long waves = ((long long)ntail * nch + slots - 1) / slots;
        const double t = (double)waves * (ch + (nch > 1 ? 8 : 0));
        if (t < best_t * 0.97) { best_t = t; best = ch; }          // prefer fewer cuts unless the gain is clear
    }
    return best;
}

// segment plan + launch of one bulk-path kernel; occs caches the kernel's resident CTAs per SM, per device (the
// shared-memory opt-in is a per-device function attribute)
constexpr int MAX_DEV = 64;
template <int DIR, bool ADV = false>
cudaError_t launch_bulk_kernel(void (*kern)(const SweepParams), int (&occs)[MAX_DEV], SweepParams& P, int sms, int user_chunk, cudaStream_t st) {
    using G = BulkGeom<DIR, ADV>;
    int dev = 0;
    cudaGetDevice(&dev);
    int& occ = occs[dev & (MAX_DEV - 1)];
    if (!occ) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)G::SMEM);
        if (e != cudaSuccess) return e;
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, G::WARPS * 32, G::SMEM);
        if (e != cudaSuccess) return e;
        if (occ < 1) occ = 1;
    }
    const int ntiles = P.ntiles, slots = sms * occ;
    if (user_chunk > 0) {                                          // explicit: every pencil in segments of user_chunk cells
        P.chunk = P.chunk_b = user_chunk;
        P.tiles_a = ntiles;
    } else {
        P.chunk = P.n;
        P.tiles_a = ntiles / slots * slots;                        // whole pencils while they fill complete waves
        P.chunk_b = (P.tiles_a < ntiles) ? ppm_tail_chunk_impl(ntiles - P.tiles_a, slots, P.n) : P.n;
    }
    const long long grid = (long long)P.tiles_a * ((P.n + P.chunk - 1) / P.chunk) + (long long)(ntiles - P.tiles_a) * ((P.n + P.chunk_b - 1) / P.chunk_b);
    kern<<<(unsigned)grid, G::WARPS * 32, G::SMEM, st>>>(P);
    return cudaGetLastError();
}
template <int DIR, int GRAV, bool FLAT>
cudaError_t launch_bulk(SweepParams& P, int sms, int user_chunk, cudaStream_t st) {
    static int occ[6][MAX_DEV] = {};
    if (P.sphere) {     // confining sphere (NEXT-3): no plane-parallel gravity, no 3-D flattening (ppm_set_sphere checks)
        if constexpr (GRAV != PPM_GRAV_CONST_Z && !FLAT) {
            if (P.cflmax) return launch_bulk_kernel<DIR>(ppm_sweep_bulk_kernel<DIR, GRAV, false, true, true, false>, occ[3], P, sms, user_chunk, st);
            return launch_bulk_kernel<DIR>(ppm_sweep_bulk_kernel<DIR, GRAV, false, false, true, false>, occ[2], P, sms, user_chunk, st);
        } else return cudaErrorNotSupported;
    }
    if (P.twof) {       // two-fluid EOS (NEXT-4): not with the 3-D flattening mode (ppm_set_two_fluid checks)
#ifndef PPM_EXP_ONE
        if constexpr (!FLAT) {
            if (P.cflmax) return launch_bulk_kernel<DIR>(ppm_sweep_bulk_kernel<DIR, GRAV, false, true, false, true>, occ[5], P, sms, user_chunk, st);
            return launch_bulk_kernel<DIR>(ppm_sweep_bulk_kernel<DIR, GRAV, false, false, false, true>, occ[4], P, sms, user_chunk, st);
        } else
#endif
        return cudaErrorNotSupported;
    }
    if (P.cflmax) return launch_bulk_kernel<DIR>(ppm_sweep_bulk_kernel<DIR, GRAV, FLAT, true, false, false>, occ[1], P, sms, user_chunk, st);
    return launch_bulk_kernel<DIR>(ppm_sweep_bulk_kernel<DIR, GRAV, FLAT, false, false, false>, occ[0], P, sms, user_chunk, st);
}
template <int DIR>
cudaError_t launch_advect_bulk(SweepParams& P, bool split, int sms, int user_chunk, cudaStream_t st) {
    static int occ[2][MAX_DEV] = {};
    if (split) return launch_bulk_kernel<DIR, true>(ppm_advect_bulk_kernel<DIR, true>, occ[1], P, sms, user_chunk, st);
    return launch_bulk_kernel<DIR>(ppm_advect_bulk_kernel<DIR, false>, occ[0], P, sms, user_chunk, st);
}
template <int DIR>
cudaError_t launch_bulk_dir(SweepParams& P, int grav, int sms, int user_chunk, cudaStream_t st) {
    const bool fl = P.flat != nullptr;
#ifdef PPM_EXP_ONE   // experiment builds: only the radial-gravity bulk sweeps are instantiated (fast compile; bench config 4/5 only)
    (void)fl; (void)grav;
    return launch_bulk<DIR, PPM_GRAV_RADIAL, false>(P, sms, user_chunk, st);
#else
    switch (grav) {
        case PPM_GRAV_NONE: return fl ? launch_bulk<DIR, PPM_GRAV_NONE, true>(P, sms, user_chunk, st) : launch_bulk<DIR, PPM_GRAV_NONE, false>(P, sms, user_chunk, st);
        case PPM_GRAV_CONST_Z: return fl ? launch_bulk<DIR, PPM_GRAV_CONST_Z, true>(P, sms, user_chunk, st) : launch_bulk<DIR, PPM_GRAV_CONST_Z, false>(P, sms, user_chunk, st);
        default: return fl ? launch_bulk<DIR, PPM_GRAV_RADIAL, true>(P, sms, user_chunk, st) : launch_bulk<DIR, PPM_GRAV_RADIAL, false>(P, sms, user_chunk, st);
    }
#endif
}

template <int DIR>
cudaError_t launch_dir(const SweepParams& P, int grav, dim3 grid, dim3 block, cudaStream_t st) {
    const bool fl = P.flat != nullptr;
#ifdef PPM_EXP_ONE
    (void)fl; (void)grav; (void)grid; (void)block; (void)st; (void)P;
    return cudaErrorNotSupported;
#else
    if (P.twof && fl) return cudaErrorNotSupported;
    switch (grav) {
        case PPM_GRAV_NONE:
            if (P.twof) ppm_sweep_kernel<DIR, PPM_GRAV_NONE, false, true><<<grid, block, 0, st>>>(P);
            else if (fl) ppm_sweep_kernel<DIR, PPM_GRAV_NONE, true, false><<<grid, block, 0, st>>>(P); else ppm_sweep_kernel<DIR, PPM_GRAV_NONE, false, false><<<grid, block, 0, st>>>(P);
            break;
        case PPM_GRAV_CONST_Z:
            if (P.twof) ppm_sweep_kernel<DIR, PPM_GRAV_CONST_Z, false, true><<<grid, block, 0, st>>>(P);
            else if (fl) ppm_sweep_kernel<DIR, PPM_GRAV_CONST_Z, true, false><<<grid, block, 0, st>>>(P); else ppm_sweep_kernel<DIR, PPM_GRAV_CONST_Z, false, false><<<grid, block, 0, st>>>(P);
            break;
        default:
            if (P.twof) ppm_sweep_kernel<DIR, PPM_GRAV_RADIAL, false, true><<<grid, block, 0, st>>>(P);
            else if (fl) ppm_sweep_kernel<DIR, PPM_GRAV_RADIAL, true, false><<<grid, block, 0, st>>>(P); else ppm_sweep_kernel<DIR, PPM_GRAV_RADIAL, false, false><<<grid, block, 0, st>>>(P);
            break;
    }
    return cudaGetLastError();
#endif
}

}  // namespace

int ppm_tail_chunk(int ntail, int slots, int n) { return ppm_tail_chunk_impl(ntail, slots, n); }

bool ppm_axis_is_bulk(const ppm_ctx* c, int axis) {
    const int ext[3] = {c->prm.nx, c->prm.ny, c->prm.nz};
    return c->io_path == 0 && ext[axis] % 4 == 0;
}

cudaError_t ppm_launch_sweep(ppm_ctx* c, int axis, double dt, bool advect, bool fuse_cfl) {
    const ppm_params& p = c->prm;
    SweepParams P;
    // A PPB-only sweep through the bulk-staged path writes the PPB part of the records only: the hydro fields stay in the buffer
    // c->hyd while the PPB coefficients move to the other one.  Every other kind of sweep needs (and leaves) a whole state.
    // (only on grids where all three axes take that path: a direct-path sweep in between would need the whole state back each time)
    const bool split = advect && ppm_axis_is_bulk(c, 0) && ppm_axis_is_bulk(c, 1) && ppm_axis_is_bulk(c, 2);
    if (!split) { cudaError_t ew = ppm_make_whole(c); if (ew != cudaSuccess) return ew; }
    P.in = c->buf[c->cur];
    P.out = c->buf[c->cur ^ 1];
    P.hdelta = split ? (long long)(c->buf[c->hyd] - c->buf[c->cur]) : 0;
    const int ext[3] = {p.nx, p.ny, p.nz};
    const int ia = (axis == 0) ? 1 : 0;       // first transverse axis
    const int ib = (axis == 2) ? 1 : 2;       // second transverse axis
    P.n = ext[axis]; P.na = ext[ia]; P.nb = ext[ib];
    const long long SB[3] = {PPM_BRICK_FLOATS, (long long)PPM_BRICK_FLOATS * c->nbx, (long long)PPM_BRICK_FLOATS * c->nbx * c->nby};
    P.SBd = SB[axis]; P.SBa = SB[ia]; P.SBb = SB[ib];
    P.nbrick_d = (P.n + 3) / 4;
    P.bc_lo = p.bc[2 * axis]; P.bc_hi = p.bc[2 * axis + 1];
    // data path: bulk-staged when the extent along the sweep axis is whole bricks, else direct
    const bool use_bulk = ppm_axis_is_bulk(c, axis);
    int chunk = c->chunk > 0 ? c->chunk : P.n;
    if (use_bulk) chunk = (chunk + 3) / 4 * 4;
    if (chunk > P.n) chunk = P.n;
    P.chunk = chunk;
    P.dt = (float)dt; P.dx = (float)p.dx; P.dtdx = (float)(dt / p.dx); P.inv_dx = (float)(1.0 / p.dx);
    P.gamma = (float)p.gamma; P.rho_floor = (float)p.rho_floor; P.p_floor = (float)p.p_floor;
    P.gp = (float)(0.5 * (p.gamma + 1.0)); P.gmg = (float)(0.5 * (p.gamma - 1.0) / p.gamma); P.g_gm1 = (float)(p.gamma / (p.gamma - 1.0)); P.hdt = (float)(0.5 * dt);
    P.tab_n = p.grav.n; P.s0 = (float)p.grav.s0; P.inv_ds = (float)(p.grav.kind != PPM_GRAV_NONE ? 1.0 / p.grav.ds : 0.0);
    P.cen_d = (float)p.grav.center[axis]; P.cen_a = (float)p.grav.center[ia]; P.cen_b = (float)p.grav.center[ib];
    P.tab = c->tab; P.tabp = c->tabp; P.tabg = c->tabg;
    P.flag = c->flag;
    P.org_d = c->org[axis]; P.org_a = c->org[ia]; P.org_b = c->org[ib];
    P.halo_lo = c->halo[axis][0]; P.halo_hi = c->halo[axis][1];
    P.HBa = PPM_BRICK_FLOATS; P.HBb = (long long)PPM_BRICK_FLOATS * ((ext[ia] + 3) / 4);    // a halo layer: [bricks along b][bricks along a] records
    { const float one = 1.0f; unsigned int b; memcpy(&b, &one, 4); P.k10 = (unsigned long long)b; }      // the f32x2 constant (1, 0)
    P.fv_shortcut = c->fv_shortcut;
    P.twof = c->twof;
    P.beta2 = (float)(1.0 / (c->twof ? c->gam_rest - 1.0 : p.gamma - 1.0));
    P.dbeta = (float)(c->twof ? 1.0 / (c->gam_tracked - 1.0) - 1.0 / (c->gam_rest - 1.0) : 0.0);
    P.sphere = c->sphere;
    if (c->sphere) {
        P.sph_dx = p.dx; P.sph_r2 = c->sph_r * c->sph_r;
        P.sph_cd = c->sph_c[axis]; P.sph_ca = c->sph_c[ia]; P.sph_cb = c->sph_c[ib];
    }
    P.cflmax = (fuse_cfl && !advect && ppm_axis_is_bulk(c, axis)) ? c->cflmax : nullptr;
    P.flat = c->flat3d ? c->F3 : nullptr;
    P.FBd = P.SBd / PPM_NFIELDS; P.FBa = P.SBa / PPM_NFIELDS; P.FBb = P.SBb / PPM_NFIELDS;
    const int nchunks = (P.n + chunk - 1) / chunk;
    const int nba = (P.na + 3) / 4, nbb = (P.nb + 3) / 4;
    cudaError_t e;
    if (use_bulk) {
        P.ntiles = ((nba + 2 * PPM_BULK_WARPS - 1) / (2 * PPM_BULK_WARPS)) * nbb;   // CTA tile = WARPS warps x 2 brick columns along a
        const int uc = c->chunk > 0 ? chunk : 0;                              // 0: whole pencils, the last wave cut to finish together
#ifndef PPM_EXP_ONE
        if (advect) {
            if (axis == 0) e = launch_advect_bulk<0>(P, split, c->sms, uc, c->stream);
            else if (axis == 1) e = launch_advect_bulk<1>(P, split, c->sms, uc, c->stream);
            else e = launch_advect_bulk<2>(P, split, c->sms, uc, c->stream);
        } else
#endif
        if (axis == 0) e = launch_bulk_dir<0>(P, p.grav.kind, c->sms, uc, c->stream);
        else if (axis == 1) e = launch_bulk_dir<1>(P, p.grav.kind, c->sms, uc, c->stream);
        else e = launch_bulk_dir<2>(P, p.grav.kind, c->sms, uc, c->stream);
    } else {
        dim3 block(PPM_CTA, 1, 1);
        dim3 grid((nba + PPM_CTA / 16 - 1) / (PPM_CTA / 16), nbb, nchunks);
#ifndef PPM_EXP_ONE
        if (advect) {
            if (axis == 0) ppm_advect_kernel<0><<<grid, block, 0, c->stream>>>(P);
            else if (axis == 1) ppm_advect_kernel<1><<<grid, block, 0, c->stream>>>(P);
            else ppm_advect_kernel<2><<<grid, block, 0, c->stream>>>(P);
            e = cudaGetLastError();
        } else
#endif
        if (axis == 0) e = launch_dir<0>(P, p.grav.kind, grid, block, c->stream);
        else if (axis == 1) e = launch_dir<1>(P, p.grav.kind, grid, block, c->stream);
        else e = launch_dir<2>(P, p.grav.kind, grid, block, c->stream);
    }
    if (e == cudaSuccess) { c->cur ^= 1; c->launches += 1; if (!split) c->hyd = c->cur; }
    return e;
}
