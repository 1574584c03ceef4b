// hydro_riemann.cuh -- Roe / HLLC / HLLE fluxes on rotated primitive states.
#pragma once
#include "hydro_math.cuh"

namespace gamer {

template <typename T> struct RoeAvg {
    T u, v, w, H, q2, a2, a, ia;   // ia = 1/a (0 if a2 <= 0)
};

template <typename T> struct Side {
    T rho, u, v, w, P, E, H;
    T m1, m2, m3;   // momenta
};

template <typename T>
__device__ __forceinline__ void make_side(const T* W, Side<T>& s, const Phys<T>& ph) {
    s.rho = W[0]; s.u = W[1]; s.v = W[2]; s.w = W[3]; s.P = W[4];
    s.m1 = s.rho * s.u; s.m2 = s.rho * s.v; s.m3 = s.rho * s.w;
    s.E = s.P * ph.inv_gm1 + T(0.5) * (s.m1 * s.u + s.m2 * s.v + s.m3 * s.w);
    s.H = (s.E + s.P) * Ops<T>::rcp(s.rho);
}

// the same from a rotated CONSERVED state (rho, m_n, m_t1, m_t2, E): one reciprocal serves the velocities and H
template <typename T>
__device__ __forceinline__ void make_side_cons(const T* U, Side<T>& s, const Phys<T>& ph) {
    s.rho = U[0]; s.m1 = U[1]; s.m2 = U[2]; s.m3 = U[3]; s.E = U[4];
    const T ir = Ops<T>::rcp(s.rho);
    s.u = s.m1 * ir; s.v = s.m2 * ir; s.w = s.m3 * ir;
    s.P = ph.gm1 * (s.E - T(0.5) * (s.m1 * s.u + s.m2 * s.v + s.m3 * s.w));
    s.H = (s.E + s.P) * ir;
}

template <typename T>
__device__ __forceinline__ void side_flux(const Side<T>& s, T* F) {
    F[0] = s.m1;
    F[1] = s.m1 * s.u + s.P;
    F[2] = s.m2 * s.u;
    F[3] = s.m3 * s.u;
    F[4] = s.u * (s.E + s.P);
}

template <typename T>
__device__ __forceinline__ void roe_average(const Side<T>& L, const Side<T>& R, RoeAvg<T>& r, const Phys<T>& ph) {
    const T wl = Ops<T>::sqrt(L.rho), wr = Ops<T>::sqrt(R.rho);
    const T id = Ops<T>::rcp(wl + wr);
    const T fl = wl * id, fr = wr * id;
    r.u = fl * L.u + fr * R.u;
    r.v = fl * L.v + fr * R.v;
    r.w = fl * L.w + fr * R.w;
    r.H = fl * L.H + fr * R.H;
    r.q2 = r.u * r.u + r.v * r.v + r.w * r.w;
    r.a2 = ph.gm1 * (r.H - T(0.5) * r.q2);
    r.ia = r.a2 > T(0) ? Ops<T>::rsqrt(r.a2) : T(0);
    r.a = r.a2 * r.ia;
}

// HLLE (Einfeldt et al. 1991)
template <typename T>
__device__ __forceinline__ void solve_hlle(const Side<T>& L, const Side<T>& R, const RoeAvg<T>& r, T* F,
                                           const Phys<T>& ph) {
    T FL[5], FR[5];
    side_flux(L, FL);
    side_flux(R, FR);
    const T cl = Ops<T>::sqrt(ph.gamma * L.P * Ops<T>::rcp(L.rho));
    const T cr = Ops<T>::sqrt(ph.gamma * R.P * Ops<T>::rcp(R.rho));
    const T bl = Ops<T>::min(r.u - r.a, L.u - cl);
    const T br = Ops<T>::max(r.u + r.a, R.u + cr);
    const T bm = Ops<T>::min(bl, T(0)), bp = Ops<T>::max(br, T(0));
    const T id = Ops<T>::rcp(bp - bm);
    const T bb = bp * bm;
    const T UL[5] = {L.rho, L.m1, L.m2, L.m3, L.E};
    const T UR[5] = {R.rho, R.m1, R.m2, R.m3, R.E};
#pragma unroll
    for (int v = 0; v < 5; ++v) F[v] = (bp * FL[v] - bm * FR[v] + bb * (UR[v] - UL[v])) * id;
}

// HLLC (Toro 2009 ch. 10) with Einfeldt's wave-speed bounds
template <typename T>
__device__ __forceinline__ void solve_hllc(const Side<T>& L, const Side<T>& R, const RoeAvg<T>& r, T* F,
                                           const Phys<T>& ph) {
    const T cl = Ops<T>::sqrt(ph.gamma * L.P * Ops<T>::rcp(L.rho));
    const T cr = Ops<T>::sqrt(ph.gamma * R.P * Ops<T>::rcp(R.rho));
    const T SL = Ops<T>::min(r.u - r.a, L.u - cl);
    const T SR = Ops<T>::max(r.u + r.a, R.u + cr);
    // branch-free: the star-region flux of the side the axis lies on is always formed; in the supersonic cases
    // (S_L >= 0: side L, S_R <= 0: side R) its correction term is switched off, which leaves F = F_K exactly
    const T ml = L.rho * (SL - L.u), mr = R.rho * (SR - R.u);
    const T SS = (R.P - L.P + L.u * ml - R.u * mr) * Ops<T>::rcp(ml - mr);
    const bool supl = SL >= T(0), supr = SR <= T(0);
    const bool left = supl || (!supr && SS >= T(0));
    const T rho = left ? L.rho : R.rho, u = left ? L.u : R.u, v = left ? L.v : R.v, w = left ? L.w : R.w;
    const T P = left ? L.P : R.P, E = left ? L.E : R.E;
    const T m1 = left ? L.m1 : R.m1, m2 = left ? L.m2 : R.m2, m3 = left ? L.m3 : R.m3;
    const T SK = left ? SL : SR;
    const T dk = SK - u;
    const T fac = rho * dk * Ops<T>::rcp(SK - SS);
    const T ir = Ops<T>::rcp(rho);
    const T es = E * ir + (SS - u) * (SS + P * ir * Ops<T>::rcp(dk));
    const T sk = (supl || supr) ? T(0) : SK;
    const T c0 = (supl || supr) ? T(0) : fac - rho, c1 = (supl || supr) ? T(0) : fac * SS - m1;
    const T c2 = (supl || supr) ? T(0) : fac * v - m2, c3 = (supl || supr) ? T(0) : fac * w - m3;
    const T c4 = (supl || supr) ? T(0) : fac * es - E;
    F[0] = m1 + sk * c0;
    F[1] = (m1 * u + P) + sk * c1;
    F[2] = m2 * u + sk * c2;
    F[3] = m3 * u + sk * c3;
    F[4] = u * (E + P) + sk * c4;
}

// Roe (1981), no entropy fix.  Returns true if remedy (i) (L104) must be taken.
// The flux is evaluated in the one-sided form  F = F_L + sum_{lambda_k<0} lambda_k alpha_k K_k  (u~ >= 0)  or
// F = F_R - sum_{lambda_k>0} lambda_k alpha_k K_k  (u~ < 0), which equals the symmetric form
// (F_L+F_R)/2 - sum |lambda_k| alpha_k K_k / 2 because F_R - F_L = sum lambda_k alpha_k K_k holds identically for
// Roe averages; only the acoustic wave on the far side of the contact can then contribute, so the dissipation
// of the three lambda = u~ waves never has to be formed.
template <typename T>
__device__ __forceinline__ bool solve_roe(const Side<T>& L, const Side<T>& R, const RoeAvg<T>& r, T* F,
                                          const Phys<T>& ph) {
    // no early exit: the flux is formed unconditionally (garbage where the solver does not apply, then replaced by
    // the caller), which leaves one branch per solve instead of three
    bool bad = !(r.a2 > T(0));
    const T d0 = R.rho - L.rho, d1 = R.m1 - L.m1, d2 = R.m2 - L.m2, d3 = R.m3 - L.m3, d4 = R.E - L.E;
    const T u = r.u, v = r.v, w = r.w, H = r.H, a = r.a;
    const T a3 = d2 - v * d0;
    const T a4 = d3 - w * d0;
    const T d5 = d4 - a3 * v - a4 * w;
    const T a2 = ph.gm1 * r.ia * r.ia * (d0 * (H - u * u) + u * d1 - d5);
    const T up = u + a, um = u - a;
    const T a1 = (d0 * up - d1 - a * a2) * (T(0.5) * r.ia);
    const T a5 = d0 - (a1 + a2);
    const T ua = u * a;
    const T Hm = H - ua, Hp = H + ua;
    // intermediate states U_L + a1 K1 and U_R - a5 K5
    {
        const T r1 = L.rho + a1, n1 = L.m1 + a1 * um, s1 = L.m2 + a1 * v, t1 = L.m3 + a1 * w, e1 = L.E + a1 * Hm;
        const T r5 = R.rho - a5, n5 = R.m1 - a5 * up, s5 = R.m2 - a5 * v, t5 = R.m3 - a5 * w, e5 = R.E - a5 * Hp;
        // P > 0  <=>  rho*E - |m|^2/2 > 0 when rho > 0
        const T p1 = r1 * e1 - T(0.5) * (n1 * n1 + s1 * s1 + t1 * t1);
        const T p5 = r5 * e5 - T(0.5) * (n5 * n5 + s5 * s5 + t5 * t5);
        bad = bad || !(r1 > T(0)) || !(r5 > T(0)) || !(p1 > T(0)) || !(p5 > T(0));
    }
    const bool pos = u >= T(0);
    const T rho = pos ? L.rho : R.rho, un = pos ? L.u : R.u, P = pos ? L.P : R.P, E = pos ? L.E : R.E;
    const T m1 = pos ? L.m1 : R.m1, m2 = pos ? L.m2 : R.m2, m3 = pos ? L.m3 : R.m3;
    (void)rho;
    const T cm = Ops<T>::min(um, T(0)) * a1, cp = Ops<T>::max(up, T(0)) * a5;
    const T cf = pos ? cm : -cp;
    const T Kn = pos ? um : up, K4 = pos ? Hm : Hp;
    F[0] = m1 + cf;
    F[1] = (m1 * un + P) + cf * Kn;
    F[2] = m2 * un + cf * v;
    F[3] = m3 * un + cf * w;
    F[4] = un * (E + P) + cf * K4;
    return bad;
}

// Exact solver ("exact solver based on Toro (2009)", reading R21): star pressure by Newton-Raphson on
// Toro's pressure function from the two-rarefaction guess, until a relative change below 1e-6 plus one more step
// (at most 30), sampling at x/t = 0, transverse velocities from the side of the contact.  Returns true when the
// data generate vacuum (Toro eq. 4.40); the caller then uses HLLE.  IEEE division / sqrt / pow throughout: this
// solver is iterative and not on the fast path.
template <typename T>
__device__ __forceinline__ void pressure_fn(T p, T rho, T pk, T ck, T gamma, T& f, T& df) {
    if (p > pk) {
        const T A = T(2) / ((gamma + T(1)) * rho), B = (gamma - T(1)) / (gamma + T(1)) * pk;
        const T q = ::sqrt(A / (p + B));
        f = (p - pk) * q;
        df = q * (T(1) - T(0.5) * (p - pk) / (B + p));
    } else {
        const T pr = p / pk;
        f = T(2) * ck / (gamma - T(1)) * (Ops<T>::pow(pr, (gamma - T(1)) / (T(2) * gamma)) - T(1));
        df = Ops<T>::pow(pr, -(gamma + T(1)) / (T(2) * gamma)) / (rho * ck);
    }
}

template <typename T>
__device__ __noinline__ bool solve_exact(const Side<T>& L, const Side<T>& R, T* F, const Phys<T>& ph) {
    const T g = ph.gamma, gm1 = g - T(1), gp1 = g + T(1), z = gm1 / (T(2) * g);
    const T cl = ::sqrt(g * L.P / L.rho), cr = ::sqrt(g * R.P / R.rho);
    const T du = R.u - L.u;
    const T num = cl + cr - T(0.5) * gm1 * du;
    if (!(num > T(0))) return true;
    const T p0 = Ops<T>::pow(num / (cl / Ops<T>::pow(L.P, z) + cr / Ops<T>::pow(R.P, z)), T(1) / z);
    T p = p0, fl, dfl, fr, dfr;
    bool extra = false;
    for (int it = 0; it < 30; ++it) {
        pressure_fn(p, L.rho, L.P, cl, g, fl, dfl);
        pressure_fn(p, R.rho, R.P, cr, g, fr, dfr);
        T pn = p - (fl + fr + du) / (dfl + dfr);
        if (!(pn > T(0))) pn = T(1e-6) * p0;
        const T change = T(2) * Ops<T>::abs(pn - p) / (pn + p);
        p = pn;
        if (extra) break;
        if (change < T(1e-6)) extra = true;
    }
    pressure_fn(p, L.rho, L.P, cl, g, fl, dfl);
    pressure_fn(p, R.rho, R.P, cr, g, fr, dfr);
    const T us = T(0.5) * (L.u + R.u) + T(0.5) * (fr - fl);
    T rho, u, P;
    const bool left = us >= T(0);
    const Side<T>& K = left ? L : R;
    const T ck = left ? cl : cr;
    const T sg = left ? T(1) : T(-1);          // mirror the right-hand formulas onto the left-hand ones
    const T uk = sg * K.u, usk = sg * us;
    if (p > K.P) {                             // shock on this side
        const T sk = uk - ck * ::sqrt(gp1 / (T(2) * g) * p / K.P + gm1 / (T(2) * g));
        if (T(0) <= sk) { rho = K.rho; u = K.u; P = K.P; }
        else { rho = K.rho * ((p / K.P + gm1 / gp1) / (gm1 / gp1 * p / K.P + T(1))); u = us; P = p; }
    } else {                                   // rarefaction on this side
        const T sh = uk - ck, st = usk - ck * Ops<T>::pow(p / K.P, z);
        if (T(0) <= sh) { rho = K.rho; u = K.u; P = K.P; }
        else if (T(0) >= st) { rho = K.rho * Ops<T>::pow(p / K.P, T(1) / g); u = us; P = p; }
        else {
            const T cf = T(2) / gp1 + gm1 / (gp1 * ck) * uk;
            rho = K.rho * Ops<T>::pow(cf, T(2) / gm1);
            u = sg * (T(2) / gp1 * (ck + T(0.5) * gm1 * uk));
            P = K.P * Ops<T>::pow(cf, T(2) * g / gm1);
        }
    }
    const T E = P / gm1 + T(0.5) * rho * (u * u + K.v * K.v + K.w * K.w);
    F[0] = rho * u;
    F[1] = rho * u * u + P;
    F[2] = rho * u * K.v;
    F[3] = rho * u * K.w;
    F[4] = u * (E + P);
    return false;
}

// Flux through a face from the two sides.  Returns true if Roe (or the exact solver) fell back to HLLE.
template <typename T, int SOLVER>
__device__ __forceinline__ bool riemann_sides(const Side<T>& L, const Side<T>& R, T* F, const Phys<T>& ph) {
    RoeAvg<T> r;
    roe_average(L, R, r, ph);
    bool fb = false;
    if (SOLVER == ROE) {
        fb = solve_roe(L, R, r, F, ph);
        if (fb) solve_hlle(L, R, r, F, ph);
    } else if (SOLVER == HLLC) {
        solve_hllc(L, R, r, F, ph);
    } else if (SOLVER == EXACT) {
        fb = solve_exact(L, R, F, ph);
        if (fb) solve_hlle(L, R, r, F, ph);
    } else {
        solve_hlle(L, R, r, F, ph);
    }
    return fb;
}

// Flux through a face from rotated CONSERVED states (rho, m_n, m_t1, m_t2, E [, s]).
template <typename T, int SOLVER, int NV>
__device__ __forceinline__ bool riemann_flux_cons(const T* UL, const T* UR, T* F, const Phys<T>& ph) {
    Side<T> L, R;
    make_side_cons(UL, L, ph);
    make_side_cons(UR, R, ph);
    const bool fb = riemann_sides<T, SOLVER>(L, R, F, ph);
    if (NV > 5) {      // every passive scalar rides the mass flux, upwinded (R12)
        const bool up = F[0] >= T(0);
        const T fq = F[0] * Ops<T>::rcp(up ? UL[0] : UR[0]);
#pragma unroll
        for (int v = 5; v < NV; ++v) F[v] = fq * (up ? UL[v] : UR[v]);
    }
    return fb;
}

// Flux through a face from rotated primitive states.  Returns true if Roe fell back to HLLE.
template <typename T, int SOLVER, int NV>
__device__ __forceinline__ bool riemann_flux(const T* WL, const T* WR, T* F, const Phys<T>& ph) {
    Side<T> L, R;
    RoeAvg<T> r;
    make_side(WL, L, ph);
    make_side(WR, R, ph);
    roe_average(L, R, r, ph);
    bool fb = false;
    if (SOLVER == ROE) {
        fb = solve_roe(L, R, r, F, ph);
        if (fb) solve_hlle(L, R, r, F, ph);
    } else if (SOLVER == HLLC) {
        solve_hllc(L, R, r, F, ph);
    } else if (SOLVER == EXACT) {
        fb = solve_exact(L, R, F, ph);
        if (fb) solve_hlle(L, R, r, F, ph);
    } else {
        solve_hlle(L, R, r, F, ph);
    }
#pragma unroll
    for (int v = 5; v < NV; ++v) F[v] = F[0] >= T(0) ? F[0] * WL[v] : F[0] * WR[v];
    return fb;
}

}  // namespace gamer
