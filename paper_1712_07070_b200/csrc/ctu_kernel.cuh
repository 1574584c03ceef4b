// ctu_kernel.cuh -- corner-transport-upwind, 6 Riemann solves per cell (Colella 1990,
// "similar to ATHENA", Stone et al. 2008; C_CFL <= 0.5, L168) as a z-streaming patch-group kernel.
//
// One CTA advances one (16 x TY x 16) column tile, marching along z.  THREAD = CELL COLUMN: thread (ci, cj) owns cell
// (ci, cj) of every plane, ci in -1..16, cj in -1..TY (the 18 x (TY+2) cells whose traced states the scheme needs).
// Everything a thread produces for its own cell lives in registers; only what a NEIGHBOUR needs goes through shared
// memory: the + states (towards the cell to the right / above) and the fluxes at the lower faces.  Two block
// barriers per plane, every exchange array single-buffered:
//
//   iteration kk   P1  z trace of plane kk+1 (own registers), first-pass z flux H*(kk+1/2) from the z+ state of plane kk
//                      (kept from the last iteration) and the new z- state;  x and y trace of plane kk, publish x+, y+   [T]
//                  -- barrier A --
//                  P2  first-pass fluxes F*(ci-1/2), G*(cj-1/2) of plane kk (left states from [T]), publish          [F1]
//                      final fluxes F(ci-1/2), G(cj-1/2) of plane kk-1 (left states from [C]), publish                [FF]
//                      next staged plane -> primitives (all threads)
//                  -- barrier B --
//                  P3  transverse correction (coefficient dt/2dh, conserved variables, R7/R8) of the six states of plane
//                      kk: x by G*, H*; y by H*, F*; z by F*, G* (upper-face fluxes from [F1]); publish corrected x+, y+ [C];
//                      final z flux at kk-1/2 from the corrected z+ of plane kk-1 (register) and z- of plane kk;
//                      update + closing step of cell (ci, cj, kk-1) from its own lower-face fluxes, the neighbours' ([FF])
//                      and the two z fluxes.
// States are carried in CONSERVED variables, rotated for their axis (rho, m_n, m_t1, m_t2, E [, s..]): the Riemann
// solver derives what it needs with one reciprocal per side, and the correction applies to them directly.
#pragma once
#include "hydro_close.cuh"

namespace gamer {

template <typename T, int RECON, int NV, int TY, bool FUSED = false> struct CtuSmem {
    using G = Geo<TY>;
    static constexpr int R = RECON == PPM ? 2 : 1;
    static constexpr int RING = 2 * R + 2;                          // planes kk+1-R .. kk+1+R, one being converted
    static constexpr int EW = 18, EH = TY + 2;
    static constexpr int NC = EW * EH;                              // cells of a plane = threads that own one
    static constexpr int NT = (NC + 31) / 32 * 32;
    static constexpr int NCP = (NC + 3) / 4 * 4;                    // exchange arrays: [Vec4 NCP | (NV-4) x NCP]
    static constexpr int RSTG = NV * (FUSED ? G::NR * FW : G::PLN); // one landing stage (fused refresh: 24-wide rows)
    static constexpr int RAW = 0;                                   // [2][RSTG]
    static constexpr int PRIM = RAW + 2 * RSTG;                     // [RING][NV][PLN]
    static constexpr int XB = NV * NCP;                             // one exchange array
    static constexpr int TX = PRIM + RING * NV * G::PLN;            // traced x+ / y+ of the plane
    static constexpr int TYY = TX + XB;
    static constexpr int F1X = TYY + XB;                            // first-pass fluxes at the lower x / y face of each cell
    static constexpr int F1Y = F1X + XB;
    static constexpr int CX = F1Y + XB;                             // corrected x+ / y+
    static constexpr int CY = CX + XB;
    static constexpr int FFX = CY + XB;                             // final fluxes at the lower x / y face
    static constexpr int FFY = FFX + XB;
    static constexpr int END = FFY + XB;
    static_assert(RSTG % 4 == 0 && (NV * G::PLN) % 4 == 0, "16-byte alignment of the Vec4 arrays");
    static constexpr size_t BYTES = 16 + (size_t)END * sizeof(T) + (FUSED ? 128 : 0);   // 2 mbarriers first, neighbour table last
};

// PLM/PPM face values of every variable of cell c along direction D, characteristic tracing over dt/2 (R7), revert of an
// unphysical pair (R8), result as CONSERVED states in the rotated order of D: um at the lower face, up at the upper one.
// CARRY (z direction, PPM, slopes limited in primitive variables): the thread traces plane after plane of its own column,
// so of the three limited slopes a plane needs two were computed for the plane below.  cs0 / csp hold the slopes of the
// cells at planes p and p+1 (rotated order) from the last call: 0 = none yet (compute all three, fill them), 1 = use them
// as the slopes of p-1 and p, compute only the one of p+1 (one shared-memory load per variable less, too).
template <typename T, int RECON, int NV, bool EXT, int PLN, int D, int CARRY = -1>
__device__ __forceinline__ void ctu_trace(const T* const* Pz, int c, T* um, T* up, const Phys<T>& ph, Counters& cnt,
                                          T* cs0 = nullptr, T* csp = nullptr) {
    constexpr int R = RECON == PPM ? 2 : 1;
    T Wr[NV], rm[NV], rp[NV], tm[NV], tp[NV];
    if (EXT && ph.char_limit) {      // slopes limited in characteristic variables (R22): all variables together
        T W5[5][NV];
#pragma unroll
        for (int m = -R; m <= R; ++m) {
            const T* q = (D == 2) ? Pz[R + m] + c : Pz[R] + c + m * (D == 0 ? 1 : NP);
#pragma unroll
            for (int k = 0; k < NV; ++k) W5[m + 2][k] = q[nat_index(D, k) * PLN];
        }
#pragma unroll
        for (int k = 0; k < NV; ++k) Wr[k] = W5[2][k];
        face_values_char<T, RECON, NV, EXT>(W5, rm, rp, ph);
    } else {
#pragma unroll
        for (int k = 0; k < NV; ++k) {      // k: position in the rotated order, v: the natural variable there
            const int v = nat_index(D, k);
            const T* q = Pz[R] + v * PLN + c;
            Wr[k] = q[0];
            if (D == 0) face_values<T, RECON, EXT, fixed_theta(EXT, RECON)>(q, 1, rm[k], rp[k], ph);
            else if (D == 1) face_values<T, RECON, EXT, fixed_theta(EXT, RECON)>(q, NP, rm[k], rp[k], ph);
            else {
                const int o = v * PLN + c;
                if (RECON == PPM && CARRY >= 0) {
                    const T l1 = Pz[R - 1][o], r1 = Pz[R + 1][o], r2 = Pz[2 * R][o];
                    T sm, s0;
                    if (CARRY == 0) {
                        const T l2 = Pz[0][o];
                        sm = limited_slope<T, EXT, fixed_theta(EXT, RECON)>(l1 - l2, Wr[k] - l1, ph);
                        s0 = limited_slope<T, EXT, fixed_theta(EXT, RECON)>(Wr[k] - l1, r1 - Wr[k], ph);
                    } else {
                        sm = cs0[k];
                        s0 = csp[k];
                    }
                    const T sp = limited_slope<T, EXT, fixed_theta(EXT, RECON)>(r1 - Wr[k], r2 - r1, ph);
                    ppm_faces<T>(l1, Wr[k], r1, sm, s0, sp, rm[k], rp[k]);
                    cs0[k] = s0;
                    csp[k] = sp;
                } else if (RECON == PPM)
                    face_values5<T, RECON, EXT>(Pz[0][o], Pz[R - 1][o], Pz[R][o], Pz[R + 1][o], Pz[2 * R][o], rm[k], rp[k], ph);
                else
                    face_values5<T, RECON, EXT>(T(0), Pz[R - 1][o], Pz[R][o], Pz[R + 1][o], T(0), rm[k], rp[k], ph);
            }
        }
    }
    trace_cell<T, RECON, NV>(Wr, rm, rp, tm, tp, ph);
    if (EXT && ph.floors) { floor_prim(tm, ph); floor_prim(tp, ph); }
    if (!(tm[0] > T(0) && tm[4] > T(0) && tp[0] > T(0) && tp[4] > T(0))) {
        cnt.reverted++;
#pragma unroll
        for (int v = 0; v < NV; ++v) { tm[v] = rm[v]; tp[v] = rp[v]; }
    }
    prim2cons<T, NV>(tm, um, ph);      // rotation commutes with the conversion: component 1 is the normal one in both
    prim2cons<T, NV>(tp, up, ph);
}

// Transverse correction of one rotated conserved state of axis D: U - dt/2dh g1 - dt/2dh g2 (g1, g2: flux differences
// across the cell along the two other axes, natural variable order); an unphysical result keeps the traced state (R8).
template <typename T, int NV, bool EXT, int D>
__device__ __forceinline__ void ctu_correct(T* U, const T* g1, const T* g2, const Phys<T>& ph, Counters& cnt) {
    T C[NV];
#pragma unroll
    for (int k = 0; k < NV; ++k) C[k] = U[k] - ph.hlam * g1[nat_index(D, k)] - ph.hlam * g2[nat_index(D, k)];
    bool ok;
    if (EXT && ph.floors) {
        T W[NV];
        cons2prim<T, NV>(C, W, ph);
        floor_prim(W, ph);
        prim2cons<T, NV>(W, C, ph);
        ok = (W[0] > T(0)) && (W[4] > T(0));
    } else {      // rho > 0 and P > 0  <=>  rho > 0 and rho E - |m|^2 / 2 > 0
        const T pe = C[0] * C[4] - T(0.5) * (C[1] * C[1] + C[2] * C[2] + C[3] * C[3]);
        ok = (C[0] > T(0)) && (pe > T(0));
    }
    if (!ok) cnt.reverted++;
#pragma unroll
    for (int k = 0; k < NV; ++k) U[k] = ok ? C[k] : U[k];
}

// one Riemann solve on rotated conserved states; flux returned in the natural variable order
template <typename T, int SOLVER, int NV, int D>
__device__ __forceinline__ void ctu_solve(const T* UL, const T* UR, T* Fnat, const Phys<T>& ph, Counters& cnt) {
    T F[NV];
    cnt.roe_fb += riemann_flux_cons<T, SOLVER, NV>(UL, UR, F, ph) ? 1 : 0;
#pragma unroll
    for (int v = 0; v < NV; ++v) Fnat[v] = F[rot_index(D, v)];
}

template <typename T, int RECON, int SOLVER, int NV, bool EXT, int TY, bool FUSED>
__global__ void __launch_bounds__((CtuSmem<T, RECON, NV, TY, FUSED>::NT), 1) ctu_kernel(const AdvArgs<T> a) {
    using G = Geo<TY>;
    using S = CtuSmem<T, RECON, NV, TY, FUSED>;
    constexpr int RS = S::RSTG, R = S::R, RING = S::RING, NT = S::NT, NC = S::NC, NCP = S::NCP;
    constexpr int NPL = 18 + 2 * R;      // staged planes: padded PF .. PF+NPL-1, staged plane n = cell plane n - 1 - R
    constexpr int PF = 2 - R;
    constexpr int PLN = G::PLN, SP = NV * G::PLN, EW = S::EW;
    constexpr int PSQ = PS * PS, PS3 = PS * PS * PS;

    extern __shared__ __align__(128) unsigned char smem_raw[];
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem_raw);
    T* sm = reinterpret_cast<T*>(smem_raw + 16);
    T* raw = sm + S::RAW;
    T* prim = sm + S::PRIM;
    T* tx = sm + S::TX;
    T* ty = sm + S::TYY;
    T* f1xs = sm + S::F1X;
    T* f1ys = sm + S::F1Y;
    T* cxs = sm + S::CX;
    T* cys = sm + S::CY;
    T* ffxs = sm + S::FFX;
    T* ffys = sm + S::FFY;

    const int tid = threadIdx.x;
    const long long tile = blockIdx.x;
    const long long g = tile / G::NTILE;
    const int j0 = (int)(tile % G::NTILE) * TY;
    // padded mode: this group's padded slab; fused mode (a.nbr set): the whole unpadded batch, ghost zones gathered
    // from the same-level neighbours inside the kernel (hydro_stream.cuh "Fused ghost refresh")
    const T* gin = FUSED ? a.in : a.in + (size_t)g * NV * NPC;
    int* nb = reinterpret_cast<int*>(smem_raw + 16 + S::END * sizeof(T));
    constexpr int NCD = FUSED ? (FusedCopies<T, NV, TY>::N + NT - 1) / NT : 1;      // fused mode: this thread's entries of the copy list
    int2 cd[NCD];
    if (FUSED) {
        if (tid < 27) nb[tid] = a.nbr[g * 27 + tid];
#pragma unroll
        for (int i = 0; i < NCD; ++i) {
            const int it = tid + i * NT;
            cd[i] = it < FusedCopies<T, NV, TY>::N ? fused_copy_desc<T, NV, TY>(it, j0) : make_int2(-1, 0);
        }
    }
    T* gout = a.out + (size_t)g * NV * PS3;
    T* gflux = a.flux ? a.flux + (size_t)g * 9 * NV * PSQ : nullptr;
    const Phys<T> ph = make_phys<T>(a);

    // ---- the cell column this thread owns.  Interior cells first, a warp holding rows w and w + TY/2 (its two 16-lane
    // halves then fall in disjoint shared-memory banks: 8 x 22 words = 16 mod 32); then the two x-halo columns
    // (ci = -1, 16, interleaved row by row), then the two y-halo rows.  Halo warps skip what only
    // interior cells do (final z solve, update) instead of idling through it in every warp.
    constexpr int NI = PS * TY, NXH = 2 * (TY + 2);
    // the x-halo threads get whole warps when the CTA has spare threads for it, so that the y-halo rows start a warp
    constexpr int XS = (NI + (NXH + 31) / 32 * 32 + 2 * PS <= NT) ? (NXH + 31) / 32 * 32 : NXH;
    bool cell = true;
    int ci = 0, cj = 0;
    if (tid < NI) {
        ci = tid & 15;
        cj = (tid >> 5) + ((tid >> 4) & 1) * (TY / 2);
    } else if (tid < NI + XS) {
        const int u = tid - NI;      // the two columns interleaved: a quarter-warp holds 4 rows x 2 columns, whose 16-byte exchange
        ci = (u & 1) ? PS : -1;      // entries (row stride 18 Vec4 = 8 banks, column offset 17 Vec4 = 4 banks) and whose
        cj = (u >> 1) - 1;           // primitive cells (row stride 22 words, column offset 17) fall on distinct banks
        cell = u < NXH;
        if (!cell) { ci = 0; cj = 0; }
    } else if (tid < NI + XS + 2 * PS) {
        const int u = tid - NI - XS;
        ci = u & 15;
        cj = u < PS ? -1 : TY;
    } else {
        cell = false;
    }
    const bool rowin = cell && cj >= 0 && cj < TY, colin = cell && ci >= 0 && ci < PS;
    // interior cells fill whole warps (NI is a multiple of 32): the flag through a warp vote is a uniform predicate
    const bool inner = __all_sync(0xffffffffu, tid < NI);
    const bool plus = rowin || colin;                                // not a corner: its z states are needed
    const bool facex = cell && ci >= 0, facey = cell && cj >= 0;     // has a lower x / y face among the 18 x (TY+2) cells
    const int c = (cj + NGH) * NP + (ci + NGH);                      // the cell inside a staged plane
    const int e = (cj + 1) * EW + (ci + 1);                          // the cell inside an exchange array
    const int gj = j0 + cj;

    if (tid == 0) {
        mbar_init(&bars[0], 1);
        mbar_init(&bars[1], 1);
        mbar_fence_init();
    }
    __syncthreads();
    auto issue = [&](int n) {      // stage padded plane PF + n into landing stage n & 1
        if (FUSED) {
            if (n < NPL) stage_plane_fused_regs<T, NV, NCD>(gin, nb, cd, PF + n, raw + (n & 1) * RS);
            else cp_async_commit();      // keeps "all but the newest group" = "everything older than one barrier"
        } else if (tid == 0 && n < NPL) {
            issue_plane<T, NV, TY>(gin, j0, PF + n, raw + (n & 1) * RS, &bars[n & 1]);
        }
    };
    auto convert = [&](int n) {    // staged plane n -> primitives of cell plane n - 1 - R, ring slot n % RING
        T* dst = prim + (n % RING) * SP;
        if (FUSED) {
            convert_plane_fused<T, NV, EXT, TY, NT>(raw + (n & 1) * RS, dst, ph, tid);
        } else {
            mbar_wait(&bars[n & 1], (n >> 1) & 1);
            convert_plane<T, NV, EXT, TY, NT>(raw + (n & 1) * RS, dst, ph, tid);
        }
    };
    issue(0);
    issue(1);
    for (int n = 0; n < RING; ++n) {      // cell planes -1-R .. R: what the z trace of planes -1 and 0 reads
        if (FUSED) { cp_async_wait<0>(); __syncthreads(); }
        convert(n);
        __syncthreads();
        issue(n + 2);
    }
    // ring slot of cell plane p (p >= -1-R)
    auto slot = [&](int p) { return ((p + 1 + R) % RING) * SP; };

    Counters cnt = {0, 0, 0, 0, 0};
    T smax = T(0);
    T zmT[NV], zpT[NV];        // traced z-, z+ of plane kk
    T hlo[NV];                 // first-pass z flux at kk-1/2 (natural order)
    T czp[NV];                 // corrected z+ of plane kk-1
    T fzlo[NV];                // final z flux at the lower face of plane kk-1
    T cxm[NV], cym[NV];        // corrected x-, y- of plane kk-1
#pragma unroll
    for (int v = 0; v < NV; ++v) { zmT[v] = zpT[v] = czp[v] = cxm[v] = cym[v] = T(1); hlo[v] = fzlo[v] = T(0); }
    // z slopes carried from plane to plane (fast kernels; the extended ones may limit in characteristic variables)
    constexpr bool ZC = RECON == PPM && !EXT;
    T zs0[NV], zsp[NV];
#pragma unroll
    for (int v = 0; v < NV; ++v) zs0[v] = zsp[v] = T(0);
    if (plus) {                // z trace of plane -1
        const T* Pz[2 * R + 1];
#pragma unroll
        for (int m = 0; m <= 2 * R; ++m) Pz[m] = prim + slot(-1 - R + m);
        ctu_trace<T, RECON, NV, EXT, PLN, 2, ZC ? 0 : -1>(Pz, c, zmT, zpT, ph, cnt, zs0, zsp);
    }

#pragma unroll 1
    for (int kk = -1; kk <= PS; ++kk) {
        const bool mid = kk >= 0 && kk < PS;
        T zmN[NV], zpN[NV], hhi[NV];           // traced z states of plane kk+1, first-pass z flux at kk+1/2
        T xm[NV], xp[NV], ym[NV], yp[NV];      // x / y states of plane kk
        // ------------------------------------------------------------------ P1
        if (kk < PS && plus) {
            const T* Pz[2 * R + 1];
#pragma unroll
            for (int m = 0; m <= 2 * R; ++m) Pz[m] = prim + slot(kk + 1 - R + m);
            ctu_trace<T, RECON, NV, EXT, PLN, 2, ZC ? 1 : -1>(Pz, c, zmN, zpN, ph, cnt, zs0, zsp);
            ctu_solve<T, SOLVER, NV, 2>(zpT, zmN, hhi, ph, cnt);
        }
        if (cell && (mid || plus)) {      // planes -1 and 16 feed the z correction of interior cells only: no corners
            const T* Pz[2 * R + 1];
#pragma unroll
            for (int m = 0; m <= 2 * R; ++m) Pz[m] = prim + slot(kk);      // in-plane stencils only
            ctu_trace<T, RECON, NV, EXT, PLN, 0>(Pz, c, xm, xp, ph, cnt);
            put_state<T, NV>(tx, NCP, e, xp);
            ctu_trace<T, RECON, NV, EXT, PLN, 1>(Pz, c, ym, yp, ph, cnt);
            put_state<T, NV>(ty, NCP, e, yp);
        }
        if (FUSED) cp_async_wait<1>();      // the plane converted below: issued two barriers ago
        __syncthreads();                    // ---- barrier A
        // ------------------------------------------------------------------ P2
        T f1x[NV], f1y[NV], ffx[NV], ffy[NV], U0[NV];
        // conserved input of cell (ci, cj, kk-1): padded mode: cell of the padded slab; fused mode: of the group's own state
        const T* gcell = FUSED ? gin + (size_t)nb[13] * NV * PS3 + (size_t)(kk - 1) * PSQ + gj * PS + ci
                               : gin + (size_t)(kk - 1 + NGH) * (NP * NP) + (gj + NGH) * NP + (ci + NGH);
        if (inner && kk >= 1) {      // loaded two phases ahead of its use
#pragma unroll
            for (int v = 0; v < NV; ++v) U0[v] = __ldg(gcell + (size_t)v * (FUSED ? PS3 : NPC));
        }
        if (facex && (mid || rowin)) {
            T UL[NV];
            get_state<T, NV>(tx, NCP, e - 1, UL);
            ctu_solve<T, SOLVER, NV, 0>(UL, xm, f1x, ph, cnt);
            put_state<T, NV>(f1xs, NCP, e, f1x);
        }
        if (facey && (mid || colin)) {
            T UL[NV];
            get_state<T, NV>(ty, NCP, e - EW, UL);
            ctu_solve<T, SOLVER, NV, 1>(UL, ym, f1y, ph, cnt);
            put_state<T, NV>(f1ys, NCP, e, f1y);
        }
        if (kk >= 1) {      // final x / y fluxes of plane kk-1 (0..15)
            if (facex && rowin) {
                T UL[NV];
                get_state<T, NV>(cxs, NCP, e - 1, UL);
                ctu_solve<T, SOLVER, NV, 0>(UL, cxm, ffx, ph, cnt);
                put_state<T, NV>(ffxs, NCP, e, ffx);
                if (gflux != nullptr && (ci & 7) == 0) {      // patch-boundary faces 0, 8, 16 (L112)
                    T* q = gflux + (size_t)((0 * 3 + (ci >> 3)) * NV) * PSQ + (kk - 1) * PS + gj;
#pragma unroll
                    for (int v = 0; v < NV; ++v) q[(size_t)v * PSQ] = ffx[v];
                }
            }
            if (facey && colin) {
                T UL[NV];
                get_state<T, NV>(cys, NCP, e - EW, UL);
                ctu_solve<T, SOLVER, NV, 1>(UL, cym, ffy, ph, cnt);
                put_state<T, NV>(ffys, NCP, e, ffy);
                if (gflux != nullptr && (gj & 7) == 0) {
                    T* q = gflux + (size_t)((1 * 3 + (gj >> 3)) * NV) * PSQ + (kk - 1) * PS + ci;
#pragma unroll
                    for (int v = 0; v < NV; ++v) q[(size_t)v * PSQ] = ffy[v];
                }
            }
        }
        const int ncv = kk + 3 + 2 * R;      // staged plane converted in this iteration: cell plane kk+2+R
        if (ncv < NPL) convert(ncv);
        __syncthreads();                    // ---- barrier B
        issue(ncv + 2);
        // ------------------------------------------------------------------ P3
        T gx[NV], gy[NV];      // first-pass flux differences across the cell (natural order)
#pragma unroll
        for (int v = 0; v < NV; ++v) gx[v] = gy[v] = T(0);
        if (colin) {
            T fu[NV];
            get_state<T, NV>(f1xs, NCP, e + 1, fu);
#pragma unroll
            for (int v = 0; v < NV; ++v) gx[v] = fu[v] - f1x[v];
        }
        if (rowin) {
            T fu[NV];
            get_state<T, NV>(f1ys, NCP, e + EW, fu);
#pragma unroll
            for (int v = 0; v < NV; ++v) gy[v] = fu[v] - f1y[v];
        }
        if (cell) {
            if (mid) {
                T gz[NV];
#pragma unroll
                for (int v = 0; v < NV; ++v) gz[v] = plus ? hhi[v] - hlo[v] : T(0);
                if (rowin) {      // x states: corrected by the y and z flux differences
                    ctu_correct<T, NV, EXT, 0>(xm, gy, gz, ph, cnt);
                    ctu_correct<T, NV, EXT, 0>(xp, gy, gz, ph, cnt);
                    put_state<T, NV>(cxs, NCP, e, xp);
                }
                if (colin) {      // y states: by z and x
                    ctu_correct<T, NV, EXT, 1>(ym, gz, gx, ph, cnt);
                    ctu_correct<T, NV, EXT, 1>(yp, gz, gx, ph, cnt);
                    put_state<T, NV>(cys, NCP, e, yp);
                }
            }
#pragma unroll
            for (int v = 0; v < NV; ++v) { cxm[v] = xm[v]; cym[v] = ym[v]; }
        }
        if (inner) {
            T fzhi[NV];
#pragma unroll
            for (int v = 0; v < NV; ++v) fzhi[v] = T(0);
            // z states of plane kk: by x and y (planes -1 .. 16)
            ctu_correct<T, NV, EXT, 2>(zmT, gx, gy, ph, cnt);
            ctu_correct<T, NV, EXT, 2>(zpT, gx, gy, ph, cnt);
            if (kk >= 0) {           // final z flux at kk-1/2
                ctu_solve<T, SOLVER, NV, 2>(czp, zmT, fzhi, ph, cnt);
                if (gflux != nullptr && (kk & 7) == 0) {
                    T* q = gflux + (size_t)((2 * 3 + (kk >> 3)) * NV) * PSQ + gj * PS + ci;
#pragma unroll
                    for (int v = 0; v < NV; ++v) q[(size_t)v * PSQ] = fzhi[v];
                }
            }
            if (kk >= 1) {           // update of cell (ci, cj, kk-1)
                const int k = kk - 1;
                T U[NV], fr[NV], fu[NV];
                get_state<T, NV>(ffxs, NCP, e + 1, fr);
                get_state<T, NV>(ffys, NCP, e + EW, fu);
#pragma unroll
                for (int v = 0; v < NV; ++v) {
                    const T dfx = fr[v] - ffx[v], dfy = fu[v] - ffy[v], dfz = fzhi[v] - fzlo[v];
                    U[v] = U0[v] - ph.lam * ((dfx + dfy) + dfz);
                }
                close_cell<T, SOLVER, NV, EXT>(U, gcell, cnt, ph);
#pragma unroll
                for (int v = 0; v < NV; ++v) gout[((size_t)v * PS + k) * PSQ + gj * PS + ci] = U[v];
                if (a.speed) {
                    const T s = signal_speed<T, NV, CTU, EXT>(U, ph);
                    smax = speed_max(smax, s);
                }
            }
#pragma unroll
            for (int v = 0; v < NV; ++v) { fzlo[v] = fzhi[v]; czp[v] = zpT[v]; }
        }
        // ------------------------------------------------------------------ plane kk+1 becomes plane kk
#pragma unroll
        for (int v = 0; v < NV; ++v) { hlo[v] = hhi[v]; zmT[v] = zmN[v]; zpT[v] = zpN[v]; }
    }

    block_epilogue<T, NT, G::NTILE, EXT>(a, g, smax, cnt, sm, tid);
}

}  // namespace gamer
