// hydro_math.cuh -- per-cell / per-face device arithmetic of the patch-group hydro solver.
// Written from the paper's method list (section 2.2) and the textbook
// formulas it names; shares nothing with oracle/ (the CPU oracle is test infrastructure).
//
// Conventions: W = primitive (rho, v0, v1, v2, P [, q]), U = conserved (rho, m0, m1, m2, E [, s]).
// "Rotated" means the face normal is component 1 (n) and the transverse ones are 2,3 (t1,t2),
// taken in cyclic order (x: y,z; y: z,x; z: x,y).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace gamer {

enum { MHM = 1, CTU = 2 };
enum { PLM = 1, PPM = 2 };
enum { ROE = 1, HLLC = 2, HLLE = 3, EXACT = 4 };
enum { LIM_GMINMOD = 1, LIM_VANLEER = 2, LIM_VANALBADA = 3 };

// ---------------------------------------------------------------------------------------------
// precision-dependent primitives.  fp32 uses the SFU approximations (<= 2 ulp); the parity bound
// of the fp32 path is 1e-5 relative L1 per step, four orders of magnitude above that.  fp64 refines
// the SFU seeds with Newton steps (<= 1.3 ulp, see Ops<double>).
// ---------------------------------------------------------------------------------------------
template <typename T> struct Ops;

template <> struct Ops<float> {
    static __device__ __forceinline__ float rcp(float x) {
        float r;
        asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
        return r;
    }
    static __device__ __forceinline__ float sqrt(float x) {
        float r;
        asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
        return r;
    }
    static __device__ __forceinline__ float rsqrt(float x) {
        float r;
        asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
        return r;
    }
    static __device__ __forceinline__ float abs(float x) { return fabsf(x); }
    static __device__ __forceinline__ float min(float a, float b) { return fminf(a, b); }
    static __device__ __forceinline__ float max(float a, float b) { return fmaxf(a, b); }
    static __device__ __forceinline__ float pow(float a, float b) { return powf(a, b); }
    static __device__ __forceinline__ float copysign(float a, float b) { return copysignf(a, b); }
    static __device__ __forceinline__ bool finite(float a) { return isfinite(a); }
    // min(|a|,|b|) if a and b have the same sign, else 0 (one FMNMX.XORSIGN + one FMNMX)
    static __device__ __forceinline__ float lo(float a, float b) { return fminf(a, b); }
    static __device__ __forceinline__ float minabs_same_sign(float a, float b) {
        float r;
        asm("min.xorsign.abs.f32 %0, %1, %2;" : "=f"(r) : "f"(a), "f"(b));
        return fmaxf(r, 0.0f);
    }
};

template <> struct Ops<double> {
    // IEEE 1.0 / x and sqrt(x) are 11 and 18 instructions with a branch to a slow path each (a fifth of the fp64 CTU
    // kernel's instructions).  These take the same SFU seed (20 bits) through branch-free Newton steps: rcp 1 ulp
    // (cubic step, 3 DFMA), sqrt 1 ulp (two coupled Goldschmidt steps), rsqrt 1.3 ulp -- measured against the IEEE
    // results over 1.3e9 arguments in 2^-20..2^20; the parity bound of the fp64 path is 1e-12.  Special values: the
    // seeds flush denormals to zero; rcp(0), rcp(inf) and sqrt(inf) return NaN instead of inf / 0 / inf (not finite
    // either way, and nothing on the path divides by an exact zero in a state that passed its positivity test);
    // sqrt(x) = 0 for |x| < DBL_MIN (sound speed at zero pressure), NaN for x < 0 like the IEEE routine.
    static __device__ __forceinline__ double rcp(double x) {
        double r;
        asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
        const double e = fma(-x, r, 1.0);
        return fma(r, fma(e, e, e), r);
    }
    static __device__ __forceinline__ double sqrt(double x) {
        double y;
        asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
        double g = x * y, h = 0.5 * y;
        double r = fma(-g, h, 0.5);
        g = fma(g, r, g);
        h = fma(h, r, h);
        r = fma(-g, h, 0.5);
        g = fma(g, r, g);
        return fabs(x) < 2.2250738585072014e-308 ? 0.0 : g;
    }
    static __device__ __forceinline__ double rsqrt(double x) {
        double y;
        asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
        double e = fma(-x * y, y, 1.0);
        y = fma(0.5 * y, e, y);
        e = fma(-x * y, y, 1.0);
        return fma(0.5 * y, e, y);
    }
    static __device__ __forceinline__ double abs(double x) { return fabs(x); }
    static __device__ __forceinline__ double min(double a, double b) { return fmin(a, b); }
    static __device__ __forceinline__ double max(double a, double b) { return fmax(a, b); }
    static __device__ __forceinline__ double pow(double a, double b) { return ::pow(a, b); }
    static __device__ __forceinline__ double copysign(double a, double b) { return ::copysign(a, b); }
    static __device__ __forceinline__ bool finite(double a) { return isfinite(a); }
    // fmin / fmax on doubles are eight instructions each (DSETP.MIN, selects, moves and the quiet-NaN fix-up); where
    // no operand can be a NaN that has to be dropped (limiter arguments) a compare + select pair does: three
    static __device__ __forceinline__ double lo(double a, double b) { return a < b ? a : b; }
    // min(|a|,|b|) if a and b have the same sign, else 0.  The sign test is taken on the sign bits as in fp32 (a zero
    // operand gives min = 0 either way; it differs from "a*b > 0" only where the product underflows)
    static __device__ __forceinline__ double minabs_same_sign(double a, double b) {
        const double m = fabs(fabs(a) < fabs(b) ? a : b);
        return (__double2hiint(a) ^ __double2hiint(b)) < 0 ? 0.0 : m;
    }
    // minmod(a, b): the one of smaller magnitude (it carries the common sign), 0 for opposite signs
    static __device__ __forceinline__ bool opposite(double a, double b) { return (__double2hiint(a) ^ __double2hiint(b)) < 0; }
    static __device__ __forceinline__ double minmag(double a, double b) { return fabs(a) < fabs(b) ? a : b; }
    static __device__ __forceinline__ double minmod(double a, double b) { return opposite(a, b) ? 0.0 : minmag(a, b); }
};

// run-time constants shared by every stage (kept in registers / constant bank)
template <typename T> struct Phys {
    T gamma, gm1, inv_gm1;
    T lam;          // dt / dh
    T hlam;         // dt / (2 dh)
    T theta;        // generalized-minmod parameter
    int limiter;    // LIM_*
    // extended mode only
    T xi, min_dens, min_pres, min_temp;
    int floors, dual, remedy2, char_limit, renorm;
};

// ---------------------------------------------------------------------------------------------
// conserved <-> primitive
// ---------------------------------------------------------------------------------------------
template <typename T, int NV>
__device__ __forceinline__ void cons2prim(const T* U, T* W, const Phys<T>& ph) {
    const T ir = Ops<T>::rcp(U[0]);
    W[0] = U[0];
    W[1] = U[1] * ir;
    W[2] = U[2] * ir;
    W[3] = U[3] * ir;
    const T ek = T(0.5) * (U[1] * W[1] + U[2] * W[2] + U[3] * W[3]);
    W[4] = ph.gm1 * (U[4] - ek);
#pragma unroll
    for (int v = 5; v < NV; ++v) W[v] = U[v] * ir;      // passive scalars: q_k = s_k / rho (L96)
}

template <typename T, int NV>
__device__ __forceinline__ void prim2cons(const T* W, T* U, const Phys<T>& ph) {
    U[0] = W[0];
    U[1] = W[0] * W[1];
    U[2] = W[0] * W[2];
    U[3] = W[0] * W[3];
    U[4] = W[4] * ph.inv_gm1 + T(0.5) * (U[1] * W[1] + U[2] * W[2] + U[3] * W[3]);
#pragma unroll
    for (int v = 5; v < NV; ++v) U[v] = W[0] * W[v];
}

template <typename T>
__device__ __forceinline__ void floor_prim(T* W, const Phys<T>& ph) {
    if (ph.min_dens > T(0) && W[0] < ph.min_dens) W[0] = ph.min_dens;
    T pf = ph.min_pres;
    const T pt = W[0] * ph.min_temp;
    if (pt > pf) pf = pt;
    if (pf > T(0) && W[4] < pf) W[4] = pf;
}

// ---------------------------------------------------------------------------------------------
// slope limiters (L94)
// ---------------------------------------------------------------------------------------------
// THETA = 1 or 2 fixes the generalized-minmod parameter at compile time (the defaults of the 11-argument form:
// 1 for PLM, 2 for PPM); THETA = 0 reads ph.theta / ph.limiter at run time (extended mode).
// The sign test "dL*dR > 0" is taken on the sign bits (min.xorsign.abs in fp32): it differs from the product
// only when the product underflows, where the slope is below 1e-19 of the data either way.
template <typename T, bool EXT, int THETA = 0>
__device__ __forceinline__ T limited_slope(T dL, T dR, const Phys<T>& ph) {
    if (THETA == 0 && EXT && ph.limiter != LIM_GMINMOD) {
        const T prod = dL * dR;
        if (!(prod > T(0))) return T(0);
        if (ph.limiter == LIM_VANLEER) return T(2) * prod * Ops<T>::rcp(dL + dR);
        return prod * (dL + dR) * Ops<T>::rcp(dL * dL + dR * dR);
    }
    if constexpr (sizeof(T) == 8) {
        // fp64 has no min/max/abs/copysign instructions: every one of them is a compare + two selects or a pair of
        // moves.  Signed form of the lines below, same values: the smaller of dL, dR carries the sign already, and
        // the centred difference has it too
        T sl = Ops<T>::minmod(dL, dR);
        if (THETA == 2 || (THETA == 0 && ph.theta != T(1))) sl = Ops<T>::minmag(THETA == 2 ? sl + sl : ph.theta * sl, T(0.5) * (dL + dR));
        return sl;
    }
    T m = Ops<T>::minabs_same_sign(dL, dR);
    // theta == 1 (plain minmod): |dL+dR|/2 >= min(|dL|,|dR|) holds exactly in floating point for equal
    // signs (rounding is monotonic), so the centred term can never win and is skipped
    if (THETA == 2) m = Ops<T>::lo(m + m, T(0.5) * Ops<T>::abs(dL + dR));
    else if (THETA == 0 && ph.theta != T(1)) m = Ops<T>::lo(ph.theta * m, T(0.5) * Ops<T>::abs(dL + dR));
    return Ops<T>::copysign(m, dR);
}

// compile-time theta of the fast (non-extended) kernels: the 11-argument defaults, theta = 1 (PLM) / 2 (PPM)
__host__ __device__ constexpr int fixed_theta(bool ext, int recon) { return ext ? 0 : (recon == PLM ? 1 : 2); }

// PPM face values of a cell from its value c, its neighbours l1, r1 and the limited slopes sm, s0, sp of the three cells
// (Colella & Woodward 1984 eqs. 1.6, 1.10)
template <typename T>
__device__ __forceinline__ void ppm_faces(T l1, T c, T r1, T sm, T s0, T sp, T& wm, T& wp) {
    const T sixth = T(1.0 / 6.0);
    const T m = T(0.5) * (l1 + c) - (s0 - sm) * sixth;
    const T p = T(0.5) * (c + r1) - (sp - s0) * sixth;
    // Monotonisation (CW84 eq. 1.10) written without branches.  With dm = c - m, dp = p - c:
    //   (p-c)(c-m) <= 0                      <=>  dm, dp of opposite sign (or one is 0)  ->  dm = dp = 0
    //   (p-m)(c-(m+p)/2) >  (p-m)^2/6        <=>  |dm| > 2|dp|                            ->  dm = 2 dp
    //   (p-m)(c-(m+p)/2) < -(p-m)^2/6        <=>  |dp| > 2|dm|                            ->  dp = 2 dm
    // i.e. dm <- sign * min(|dm|, 2|dp|), dp <- sign * min(|dp|, 2|dm|), both 0 for opposite signs.
    const T dm = c - m, dp = p - c;
    if constexpr (sizeof(T) == 8) {      // signed form (see limited_slope): one sign test serves both faces
        const bool opp = Ops<T>::opposite(dm, dp);
        wm = c - (opp ? T(0) : Ops<T>::minmag(dm, dp + dp));
        wp = c + (opp ? T(0) : Ops<T>::minmag(dp, dm + dm));
        return;
    }
    const T am = Ops<T>::minabs_same_sign(dm, dp + dp);
    const T ap = Ops<T>::minabs_same_sign(dp, dm + dm);
    wm = c - Ops<T>::copysign(am, dm);
    wp = c + Ops<T>::copysign(ap, dp);
}

// face values of the centre cell of a strip: q points at the centre, neighbours at q[+-s], q[+-2s]
template <typename T, int RECON, bool EXT, int THETA = 0>
__device__ __forceinline__ void face_values(const T* q, int s, T& wm, T& wp, const Phys<T>& ph) {
    const T c = q[0], l1 = q[-s], r1 = q[s];
    if (RECON == PLM) {
        const T sl = limited_slope<T, EXT, THETA>(c - l1, r1 - c, ph);
        wm = c - T(0.5) * sl;
        wp = c + T(0.5) * sl;
    } else {   // PPM, Colella & Woodward (1984) eqs. 1.6-1.10, no steepening / flattening
        const T l2 = q[-2 * s], r2 = q[2 * s];
        const T sm = limited_slope<T, EXT, THETA>(l1 - l2, c - l1, ph);
        const T s0 = limited_slope<T, EXT, THETA>(c - l1, r1 - c, ph);
        const T sp = limited_slope<T, EXT, THETA>(r1 - c, r2 - r1, ph);
        ppm_faces<T>(l1, c, r1, sm, s0, sp, wm, wp);
    }
}

// ---------------------------------------------------------------------------------------------
// slope limiting in characteristic variables (L94; DESIGN R22): rotated primitive states of cells j-1, j, j+1 ->
// slope vector of cell j = R . limiter(L (W_j - W_j-1), L (W_j+1 - W_j)), eigenvectors evaluated at cell j
// ---------------------------------------------------------------------------------------------
template <typename T, int NV, bool EXT>
__device__ __forceinline__ void char_slope(const T* Wl, const T* Wc, const T* Wr, T* slope, const Phys<T>& ph) {
    const T rho = Wc[0];
    const T c2 = ph.gamma * Wc[4] / rho;
    const T cs = ::sqrt(c2);
    T aL[NV], aR[NV];
    {
        const T d0 = Wc[0] - Wl[0], d1 = Wc[1] - Wl[1], d4 = Wc[4] - Wl[4];
        aL[0] = (d4 - rho * cs * d1) / (T(2) * c2); aL[1] = d0 - d4 / c2; aL[2] = Wc[2] - Wl[2]; aL[3] = Wc[3] - Wl[3];
        aL[4] = (d4 + rho * cs * d1) / (T(2) * c2);
#pragma unroll
        for (int v = 5; v < NV; ++v) aL[v] = Wc[v] - Wl[v];
    }
    {
        const T d0 = Wr[0] - Wc[0], d1 = Wr[1] - Wc[1], d4 = Wr[4] - Wc[4];
        aR[0] = (d4 - rho * cs * d1) / (T(2) * c2); aR[1] = d0 - d4 / c2; aR[2] = Wr[2] - Wc[2]; aR[3] = Wr[3] - Wc[3];
        aR[4] = (d4 + rho * cs * d1) / (T(2) * c2);
#pragma unroll
        for (int v = 5; v < NV; ++v) aR[v] = Wr[v] - Wc[v];
    }
    T s[NV];
#pragma unroll
    for (int a = 0; a < NV; ++a) s[a] = limited_slope<T, EXT, 0>(aL[a], aR[a], ph);
    slope[0] = (s[0] + s[1]) + s[4];
    slope[1] = s[4] * cs / rho - s[0] * cs / rho;
    slope[2] = s[2];
    slope[3] = s[3];
    slope[4] = s[0] * cs * cs + s[4] * cs * cs;
#pragma unroll
    for (int v = 5; v < NV; ++v) slope[v] = s[v];
}

// face values of cell j from the rotated primitive states Wr[0..4] = cells j-2 .. j+2 (PLM reads 1..3 only)
template <typename T, int RECON, int NV, bool EXT>
__device__ __forceinline__ void face_values_char(const T (*Wr)[NV], T* rm, T* rp, const Phys<T>& ph) {
    if (RECON == PLM) {
        T sl[NV];
        char_slope<T, NV, EXT>(Wr[1], Wr[2], Wr[3], sl, ph);
#pragma unroll
        for (int v = 0; v < NV; ++v) { rm[v] = Wr[2][v] - T(0.5) * sl[v]; rp[v] = Wr[2][v] + T(0.5) * sl[v]; }
    } else {
        T sm[NV], s0[NV], sp[NV];
        char_slope<T, NV, EXT>(Wr[0], Wr[1], Wr[2], sm, ph);
        char_slope<T, NV, EXT>(Wr[1], Wr[2], Wr[3], s0, ph);
        char_slope<T, NV, EXT>(Wr[2], Wr[3], Wr[4], sp, ph);
        const T sixth = T(1.0 / 6.0);
#pragma unroll
        for (int v = 0; v < NV; ++v) {
            const T c = Wr[2][v];
            const T m = T(0.5) * (Wr[1][v] + c) - (s0[v] - sm[v]) * sixth;
            const T p = T(0.5) * (c + Wr[3][v]) - (sp[v] - s0[v]) * sixth;
            const T dm = c - m, dp = p - c;      // monotonisation as in face_values
            const T am = Ops<T>::minabs_same_sign(dm, dp + dp);
            const T ap = Ops<T>::minabs_same_sign(dp, dm + dm);
            rm[v] = c - Ops<T>::copysign(am, dm);
            rp[v] = c + Ops<T>::copysign(ap, dp);
        }
    }
}

// physical flux along axis D of a state known as W and U, added with sign sg into acc
template <typename T, int NV, int D>
__device__ __forceinline__ void phys_flux(const T* W, const T* U, T* F) {
    const T vn = W[1 + D];
    F[0] = U[0] * vn;
    F[1] = U[1] * vn;
    F[2] = U[2] * vn;
    F[3] = U[3] * vn;
    F[1 + D] += W[4];
    F[4] = vn * (U[4] + W[4]);
#pragma unroll
    for (int v = 5; v < NV; ++v) F[v] = U[v] * vn;
}

// ---------------------------------------------------------------------------------------------
// CTU characteristic tracing over dt/2 (Colella 1990; Colella & Woodward 1984 eq. 1.12): rotated
// primitive cell value W and untraced face values wm/wp -> traced tm/tp.  Reference state = average
// over the domain of dependence of the fastest wave toward the face; the slower waves that also
// move toward the face are corrected to their own domains.
// ---------------------------------------------------------------------------------------------
template <typename T, int RECON, int NV>
__device__ __forceinline__ void trace_cell(const T* W, const T* wm, const T* wp, T* tm, T* tp,
                                           const Phys<T>& ph) {
    const T rho = W[0], vn = W[1];
    const T c2 = ph.gamma * W[4] * Ops<T>::rcp(rho);
    const T cs = Ops<T>::sqrt(c2);
    const T l1 = vn - cs, l5 = vn + cs;
    const T x1 = l1 * ph.lam, x0 = vn * ph.lam, x5 = l5 * ph.lam;
    const T x5p = x5 > T(0) ? x5 : T(0);
    const T x1m = x1 < T(0) ? x1 : T(0);
    const T third = T(1.0 / 3.0);
    T d[NV], w6[NV];
#pragma unroll
    for (int v = 0; v < NV; ++v) {
        d[v] = wp[v] - wm[v];
        w6[v] = RECON == PPM ? T(6) * (W[v] - T(0.5) * (wm[v] + wp[v])) : T(0);
        tp[v] = wp[v] - T(0.5) * x5p * (d[v] - (T(1) - T(2) * third * x5p) * w6[v]);
        tm[v] = wm[v] - T(0.5) * x1m * (d[v] + (T(1) + T(2) * third * x1m) * w6[v]);
    }
    const T ic2 = Ops<T>::rcp(c2);
    const T rc = rho * cs;
    const T cor = cs * Ops<T>::rcp(rho);
    // ---- plus face: waves with lambda > 0
    if (l1 > T(0)) {
        const T A = T(0.5) * (x5p - x1), B = third * (x5p * x5p - x1 * x1);
        const T vP = A * (d[4] - w6[4]) + B * w6[4];
        const T vU = A * (d[1] - w6[1]) + B * w6[1];
        const T amp = (vP - rc * vU) * (T(0.5) * ic2);
        tp[0] += amp;
        tp[1] -= amp * cor;
        tp[4] += amp * c2;
    }
    {   // the lambda = vn waves reach one face or the other in every cell, and neighbouring cells disagree: taken without a
        // branch (zero coefficients on the far face); the acoustic corrections above and below apply to supersonic cells only
        const bool on = vn > T(0);
        const T A = on ? T(0.5) * (x5p - x0) : T(0), B = on ? third * (x5p * x5p - x0 * x0) : T(0);
        const T vR = A * (d[0] - w6[0]) + B * w6[0];
        const T vP = A * (d[4] - w6[4]) + B * w6[4];
        tp[0] += vR - vP * ic2;
        tp[2] += A * (d[2] - w6[2]) + B * w6[2];
        tp[3] += A * (d[3] - w6[3]) + B * w6[3];
#pragma unroll
        for (int v = 5; v < NV; ++v) tp[v] += A * (d[v] - w6[v]) + B * w6[v];
    }
    // ---- minus face: waves with lambda < 0
    if (l5 < T(0)) {
        const T C = T(0.5) * (x1m - x5), D = third * (x1m * x1m - x5 * x5);
        const T vP = C * (d[4] + w6[4]) + D * w6[4];
        const T vU = C * (d[1] + w6[1]) + D * w6[1];
        const T amp = (vP + rc * vU) * (T(0.5) * ic2);
        tm[0] += amp;
        tm[1] += amp * cor;
        tm[4] += amp * c2;
    }
    {
        const bool on = vn < T(0);
        const T C = on ? T(0.5) * (x1m - x0) : T(0), D = on ? third * (x1m * x1m - x0 * x0) : T(0);
        const T vR = C * (d[0] + w6[0]) + D * w6[0];
        const T vP = C * (d[4] + w6[4]) + D * w6[4];
        tm[0] += vR - vP * ic2;
        tm[2] += C * (d[2] + w6[2]) + D * w6[2];
        tm[3] += C * (d[3] + w6[3]) + D * w6[3];
#pragma unroll
        for (int v = 5; v < NV; ++v) tm[v] += C * (d[v] + w6[v]) + D * w6[v];
    }
}

}  // namespace gamer
