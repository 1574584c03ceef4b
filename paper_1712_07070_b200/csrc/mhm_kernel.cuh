// mhm_kernel.cuh -- MUSCL-Hancock (MHM; Toro 2009 sect. 14.4/16.5) patch-group kernel.
//
// One CTA advances one (16 x TY x 16) column tile of a patch group, marching along z, ONE block barrier
// per plane.  Thread roles (fixed for the whole kernel):
//   interior (16*TY threads) : cell (i, j) of the tile.  Per plane kk it runs the predictor of its cell
//        (PLM/PPM face values, Hancock half step, R6 of DESIGN.md), keeps the z+ / z- states and the
//        x-, y- states in registers, publishes only x+ and y+ to shared memory, and solves the three
//        Riemann problems at its own lower faces (i-1/2, j-1/2, kk-1/2).  It finishes cell (i, j, kk-1)
//        from registers plus the two neighbour fluxes (i+1/2, j+1/2) read from shared memory.
//   x-halo (2*TY threads)    : cells (-1, j) [publish x+] and (16, j) [solve face 15 1/2].
//   y-halo (32 threads)      : cells (i, -1) [publish y+] and (i, TY) [solve face TY - 1/2].
//   halo warps also turn each staged conserved plane (TMA 1-D bulk copies, two stages) into primitives
//   in a ring of 2R+2 planes, one plane ahead of the predictor.
// Face states and fluxes in shared memory are double-buffered by plane parity, which is what lets a
// single __syncthreads per plane separate "publish" from "consume":
//   iteration kk:  predictor(kk), z-Riemann(kk-1/2), convert(plane kk+2+R)  | barrier |
//                  x/y-Riemann(kk), update of plane kk-1, TMA issue for the freed stage.
// All threads run the same loop body (one copy of the predictor and of each of the three Riemann solves, so
// the code stays inside the 32 KB instruction cache and a face shared by two groups gets bit-identical
// fluxes from both); roles only switch parts of it off.
#pragma once
#include "hydro_close.cuh"


namespace gamer {

template <typename T, int RECON, int NV, int TY, int NSTG = 2, bool FUSED = false, bool VLS = false> struct MhmGeo {
    static constexpr int R = RECON == PPM ? 2 : 1;
    static constexpr int RSTAGE = VLS ? R + 1 : R;              // planes staged beyond the tile: the VL half-step predictor reaches one cell further
    static constexpr int RING = 2 * R + 2;
    static constexpr int NI = 16 * TY;                          // interior threads
    static constexpr int NXH = 2 * TY, NYH = 32;                // halo threads
    static constexpr int NT = ((NI + NXH + NYH + 31) / 32) * 32;
    static constexpr int NCV = NT - NI;                         // threads that convert planes
    static constexpr int NTILE = PS / TY;
    static constexpr int NR = TY + 2 * NGH, PLN = NR * NP;      // staged plane
    // row stride of the exchange arrays: 18 entries (17 x faces / 16 y faces used).  A warp holds rows w and w + TY/2; with
    // 8 * 18 = 16 mod 32 the scalar fifth components of its two half-warps fall on disjoint banks (17 and 16 gave 2-way conflicts)
    static constexpr int SW = 18;
    static constexpr int NSX = (SW * TY + 3) / 4 * 4, NSY = (SW * (TY + 1) + 3) / 4 * 4;     // x+ states / x fluxes, y+ states / y fluxes
    static constexpr int BLK = (NSX + NSY) * NV;                // one buffer of states (or of fluxes)
    static constexpr int RSTG = NV * (FUSED ? NR * FW : PLN);   // one landing stage (fused refresh: 24-wide rows)
    static constexpr int RAW = 0;                               // [NSTG][RSTG]  TMA / cp.async landing stages
    static constexpr int PRIM = RAW + NSTG * RSTG;              // [RING][NV][PLN]  (VL: primitives of the half-step state)
    static constexpr int ST = PRIM + RING * NV * PLN;           // [2] x [Vec4 NSX | (NV-4) NSX | Vec4 NSY | (NV-4) NSY]
    static constexpr int FL = ST + 2 * BLK;                     // same shape, fluxes in natural variable order
    static constexpr int END0 = FL + 2 * BLK;
    // VL scheme only: primitives of U^n (3 planes) and the first-order fluxes of the half-step predictor, [NV][n] each
    static constexpr int NRH = TY + 4;                          // rows of half-step cells: -2 .. TY+1
    static constexpr int NF1X = 21 * NRH, NF1Y = 20 * (NRH + 1), NF1Z = 20 * NRH;
    static constexpr int WN = END0;                             // [3][NV][PLN]
    static constexpr int F1X = WN + 3 * NV * PLN;
    static constexpr int F1Y = F1X + NV * NF1X;
    static constexpr int F1Z = F1Y + NV * NF1Y;                 // [2][NV][NF1Z]: faces below planes of even / odd padded index
    static constexpr int END = VLS ? F1Z + 2 * NV * NF1Z : END0;
    static constexpr int NCOPY = FUSED ? FusedCopies<T, NV, TY>::N : 0;                   // fused refresh: copy list
    static constexpr size_t BYTES = 16 + (size_t)END * sizeof(T) + (FUSED ? 128 : 0);   // 2 mbarriers first; neighbour table last
    static_assert((NV * PLN) % 4 == 0 && NSX % 4 == 0 && NSY % 4 == 0, "16-byte alignment of the Vec4 arrays");
};

// ---------------------------------------------------------------------------------------------
// predictor pieces (DESIGN R6)
// ---------------------------------------------------------------------------------------------
// Face values of one cell in all three directions -> conserved face states Uf[d][s] and the sum over d of
// F_d(W+) - F_d(W-).  Pz[m] points at variable 0 of this cell in the primitive plane kk-R+m.
// Packed form (fp32, Blackwell fma.rn.f32x2): the minus and plus state of one direction evolved and tested together,
// two FMAs per instruction.  Same arithmetic per lane as mhm_evolve.
__device__ __forceinline__ uint64_t pk2(float a, float b) { uint64_t r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b)); return r; }
__device__ __forceinline__ void upk2(uint64_t r, float& a, float& b) { asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(r)); }
__device__ __forceinline__ uint64_t fma2(uint64_t a, uint64_t b, uint64_t c) { uint64_t r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
__device__ __forceinline__ uint64_t mul2(uint64_t a, uint64_t b) { uint64_t r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }

template <typename T, int RECON, int NV, bool EXT, int PLN>
__device__ __forceinline__ void mhm_face_states(const T* const* Pz, const Phys<T>& ph, T (&Uf)[3][2][NV], T (&dU)[NV]) {
    constexpr int R = RECON == PPM ? 2 : 1;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        T Wm[NV], Wp[NV];
        if (EXT && ph.char_limit) {      // slopes limited in characteristic variables (R22): all variables together
            T Wr[5][NV], rm[NV], rp[NV];
#pragma unroll
            for (int m = -R; m <= R; ++m) {
                const T* q = (d == 2) ? Pz[R + m] : Pz[R] + m * (d == 0 ? 1 : NP);
#pragma unroll
                for (int k = 0; k < NV; ++k) Wr[m + 2][k] = q[nat_index(d, k) * PLN];
            }
            face_values_char<T, RECON, NV, EXT>(Wr, rm, rp, ph);
#pragma unroll
            for (int k = 0; k < NV; ++k) { Wm[nat_index(d, k)] = rm[k]; Wp[nat_index(d, k)] = rp[k]; }
        } else
#pragma unroll
        for (int v = 0; v < NV; ++v) {
            const T* q = Pz[R] + v * PLN;
            if (d == 0) face_values<T, RECON, EXT, fixed_theta(EXT, RECON)>(q, 1, Wm[v], Wp[v], ph);
            else if (d == 1) face_values<T, RECON, EXT, fixed_theta(EXT, RECON)>(q, NP, Wm[v], Wp[v], ph);
            else {
                const int o = v * PLN;
                if (RECON == PPM)
                    face_values5<T, RECON, EXT>(Pz[0][o], Pz[R - 1][o], Pz[R][o], Pz[R + 1][o], Pz[2 * R][o], Wm[v], Wp[v], ph);
                else
                    face_values5<T, RECON, EXT>(T(0), Pz[R - 1][o], Pz[R][o], Pz[R + 1][o], T(0), Wm[v], Wp[v], ph);
            }
        }
        prim2cons<T, NV>(Wm, Uf[d][0], ph);
        prim2cons<T, NV>(Wp, Uf[d][1], ph);
        // dU += F_d(W+) - F_d(W-), accumulated term by term with fused multiply-adds
        const T vm = Wm[1 + d], vp = Wp[1 + d];
        {
            const T dm = Uf[d][1][1 + d] - Uf[d][0][1 + d];      // mass flux = momentum along d
            dU[0] = (d == 0) ? dm : dU[0] + dm;
        }
#pragma unroll
        for (int v = 1; v < NV; ++v) {
            const T am = (v == 4) ? Uf[d][0][4] + Wm[4] : Uf[d][0][v];
            const T ap = (v == 4) ? Uf[d][1][4] + Wp[4] : Uf[d][1][v];
            T acc = (d == 0) ? ap * vp : dU[v] + ap * vp;
            acc = acc - am * vm;
            dU[v] = acc;
        }
        dU[1 + d] += Wp[4] - Wm[4];
    }
}

// Hancock half step of one conserved face state: Ue = Uf - hl * dU (hl = dt/(2 dh), or 0 in the reverting pass,
// where the un-evolved face values are taken as they are); returns whether rho and P of the result are positive.
// The evolved state stays in conserved variables all the way to the Riemann solver, which derives the velocities,
// P and H it needs from them with one reciprocal (make_side_cons): no conserved -> primitive -> conserved round
// trip per state.  P > 0 is tested without a division: for rho > 0, P > 0 <=> rho E - |m|^2 / 2 > 0.
// With floors (extended mode) the state goes through primitives, as in the oracle: floor, back to conserved.
// Every thread evolves all six states of its cell, also the ones it hands to no Riemann solver: any bad state
// reverts the cell (R6) and the halo copy of a cell must decide exactly as its owner in the neighbouring group does.
template <typename T, int NV, bool EXT>
__device__ __forceinline__ bool mhm_evolve(const T* Uf, const T* dU, T hl, T* Ue, bool floors, const Phys<T>& ph) {
#pragma unroll
    for (int v = 0; v < NV; ++v) Ue[v] = Uf[v] - hl * dU[v];      // one FMA per component
    if (EXT && ph.floors && floors) {
        T We[NV];
        cons2prim<T, NV>(Ue, We, ph);
        floor_prim(We, ph);
        prim2cons<T, NV>(We, Ue, ph);
        return (We[0] > T(0)) && (We[4] > T(0));
    }
    const T pe = Ue[0] * Ue[4] - T(0.5) * (Ue[1] * Ue[1] + Ue[2] * Ue[2] + Ue[3] * Ue[3]);
    return (Ue[0] > T(0)) && (pe > T(0));
}

// (packed helpers pk2 / upk2 / fma2 / mul2: above mhm_face_states)
template <int NV>
__device__ __forceinline__ bool mhm_evolve_pair(const float* UfA, const float* UfB, const float* dU, float hl, float* UeA, float* UeB) {
    const uint64_t mh = pk2(-hl, -hl);
    uint64_t e[NV];
#pragma unroll
    for (int v = 0; v < NV; ++v) e[v] = fma2(mh, pk2(dU[v], dU[v]), pk2(UfA[v], UfB[v]));
    uint64_t q = mul2(e[1], e[1]);
    q = fma2(e[2], e[2], q);
    q = fma2(e[3], e[3], q);
    const uint64_t pe = fma2(pk2(-0.5f, -0.5f), q, mul2(e[0], e[4]));
#pragma unroll
    for (int v = 0; v < NV; ++v) upk2(e[v], UeA[v], UeB[v]);
    float pa, pb;
    upk2(pe, pa, pb);
    return (UeA[0] > 0.f) && (UeB[0] > 0.f) && (pa > 0.f) && (pb > 0.f);
}

// ---------------------------------------------------------------------------------------------
// VL scheme (DESIGN R26): the half-step predictor is a first-order Godunov update of the cell
// averages.  Two cooperative stages per plane, work items spread over all threads of the tile:
//   vl_faces : first-order fluxes from the piecewise-constant primitives W^n -- x and y faces of padded plane pm and
//              the z faces between planes pm and pm+1 -- on the 20 x (TY+4) cells the reconstruction will read;
//   vl_cells : U^{n+1/2} = U^n - dt/(2 dh) sum_d dF1_d  ->  primitives (floors; an unphysical state falls back to
//              W^n) into the ring of half-step primitive planes, which the PLM face values are then taken from.
// ---------------------------------------------------------------------------------------------
template <typename T, int SOLVER, int NV, class G, int NT>
__device__ __forceinline__ void vl_faces(const T* wlo, const T* whi, T* f1x, T* f1y, T* f1z, bool xy, const Phys<T>& ph, int tid,
                                         Counters& cnt) {
    constexpr int PLN = G::PLN, NX = G::NF1X, NY = G::NF1Y, NZ = G::NF1Z;
    for (int it = (xy ? 0 : NX + NY) + tid; it < NX + NY + NZ; it += NT) {
        int d, l, rr, n, o;
        const T* pr = wlo;
        T* fo;
        if (it < NX) {                    // x face ii (between staged columns ii, ii+1) of half-step row r
            const int r = it / 21, ii = it - r * 21;
            d = 0; l = (r + 1) * NP + ii; rr = l + 1; fo = f1x; n = NX; o = it;
        } else if (it < NX + NY) {        // y face between staged rows r, r+1, column ii+1
            const int g = it - NX;
            const int r = g / 20, ii = g - r * 20;
            d = 1; l = r * NP + ii + 1; rr = l + NP; fo = f1y; n = NY; o = g;
        } else {                          // z face between the two planes
            const int g = it - NX - NY;
            const int r = g / 20, ii = g - r * 20;
            d = 2; l = (r + 1) * NP + ii + 1; rr = l; pr = whi; fo = f1z; n = NZ; o = g;
        }
        const int cn = 1 + d, c1 = d == 2 ? 1 : 2 + d, c2 = d == 0 ? 3 : d;      // 1 + (d+1)%3, 1 + (d+2)%3
        T WL[NV], WR[NV], F[NV];
        WL[0] = wlo[l]; WL[1] = wlo[cn * PLN + l]; WL[2] = wlo[c1 * PLN + l]; WL[3] = wlo[c2 * PLN + l]; WL[4] = wlo[4 * PLN + l];
        WR[0] = pr[rr]; WR[1] = pr[cn * PLN + rr]; WR[2] = pr[c1 * PLN + rr]; WR[3] = pr[c2 * PLN + rr]; WR[4] = pr[4 * PLN + rr];
#pragma unroll
        for (int v = 5; v < NV; ++v) { WL[v] = wlo[v * PLN + l]; WR[v] = pr[v * PLN + rr]; }
        cnt.roe_fb += riemann_flux<T, SOLVER, NV>(WL, WR, F, ph) ? 1 : 0;
        fo[o] = F[0]; fo[cn * n + o] = F[1]; fo[c1 * n + o] = F[2]; fo[c2 * n + o] = F[3]; fo[4 * n + o] = F[4];
#pragma unroll
        for (int v = 5; v < NV; ++v) fo[v * n + o] = F[v];
    }
}

template <typename T, int NV, bool EXT, class G, int NT>
__device__ __forceinline__ void vl_cells(const T* wn, const T* f1x, const T* f1y, const T* fzlo, const T* fzhi, T* wh,
                                         const Phys<T>& ph, int tid, Counters& cnt) {
    constexpr int PLN = G::PLN, NX = G::NF1X, NY = G::NF1Y, NZ = G::NF1Z;
    for (int c = tid; c < NZ; c += NT) {
        const int r = c / 20, ii = c - r * 20;
        const int s = (r + 1) * NP + ii + 1;
        T W0[NV], U[NV], W[NV];
#pragma unroll
        for (int v = 0; v < NV; ++v) W0[v] = wn[v * PLN + s];
        prim2cons<T, NV>(W0, U, ph);
#pragma unroll
        for (int v = 0; v < NV; ++v) {
            const T dfx = f1x[v * NX + r * 21 + ii + 1] - f1x[v * NX + r * 21 + ii];
            const T dfy = f1y[v * NY + (r + 1) * 20 + ii] - f1y[v * NY + r * 20 + ii];
            const T dfz = fzhi[v * NZ + c] - fzlo[v * NZ + c];
            U[v] = U[v] - ph.hlam * ((dfx + dfy) + dfz);
        }
        cons2prim<T, NV>(U, W, ph);
        if (EXT && ph.floors) floor_prim(W, ph);
        const bool ok = (W[0] > T(0)) && (W[4] > T(0));
        if (!ok) cnt.reverted++;
#pragma unroll
        for (int v = 0; v < NV; ++v) wh[v * PLN + s] = ok ? W[v] : W0[v];
    }
}

// per-thread constants of the cell column this thread owns
template <typename T> struct MhmCell {
    int cidx;            // cell inside a staged plane
    int sx_own, sy_own;  // slot of the x+ (y+) state of the left (lower) neighbour = slot of the own lower-face flux
    int gin_off;         // padded cell (ei, ej, interior plane 0) of variable 0, relative to the group's `in`
    int out_off;         // cell (ei, ej) inside a 16 x 16 plane of `out` (also of a z plane of flux_out)
};

template <typename T, int RECON, int SOLVER, int NV, bool EXT, int TY, int NSTG, int MINB, bool FUSED, bool VLS>
__global__ void __launch_bounds__((MhmGeo<T, RECON, NV, TY, NSTG, FUSED, VLS>::NT), MINB) mhm_kernel(const AdvArgs<T> a) {
    using G = MhmGeo<T, RECON, NV, TY, NSTG, FUSED, VLS>;
    constexpr int RS = G::RSTG;
    constexpr int R = G::R, RING = G::RING, NT = G::NT, NI = G::NI, PLN = G::PLN, S = NV * G::PLN;
    constexpr int NPL = 18 + 2 * G::RSTAGE;      // staged planes: padded PF .. PF+NPL-1
    constexpr int PF = 2 - G::RSTAGE;
    constexpr int CV = VLS ? 7 : 2 + 2 * R;      // staged plane kk+CV is converted in iteration kk
    static_assert(!VLS || RECON == PLM, "VL + PPM would need a fourth ghost zone");
    constexpr int PSQ = PS * PS;

    extern __shared__ __align__(128) unsigned char smem_raw[];
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem_raw);
    T* sm = reinterpret_cast<T*>(smem_raw + 16);
    T* raw = sm + G::RAW;
    T* prim = sm + G::PRIM;

    const int tid = threadIdx.x;
    const long long tile = blockIdx.x;
    const long long g = tile / G::NTILE;
    const int j0 = (int)(tile % G::NTILE) * TY;
    // padded mode: this group's padded slab; fused mode: the whole unpadded batch (neighbours are read too)
    const T* gin = FUSED ? a.in : a.in + (size_t)g * NV * NPC;
    int* nb = reinterpret_cast<int*>(smem_raw + 16 + G::END * sizeof(T));      // fused mode: 27 neighbour groups
    constexpr int NCP = FUSED ? (G::NCOPY + NT - 1) / NT : 1;      // fused mode: this thread's entries of the copy list, in registers
    int2 cd[NCP];
    if (FUSED) {
        if (tid < 27) nb[tid] = a.nbr[g * 27 + tid];
#pragma unroll
        for (int i = 0; i < NCP; ++i) {
            const int it = tid + i * NT;
            cd[i] = it < G::NCOPY ? fused_copy_desc<T, NV, TY>(it, j0) : make_int2(-1, 0);
        }
    }
    const Phys<T> ph = make_phys<T>(a);

    // ---- role of this thread: cell (ei, ej) of the tile, ei in -1..16, ej in -1..TY
    // role: 0 = interior, 1 = x-low, 2 = x-high, 4 = y-low, 8 = y-high, 16 = padding thread (conversion only)
    // NI is a multiple of 32: a warp is all interior or all halo.  Taking the flag through a warp vote tells the compiler so
    // (uniform predicate, plain branches without convergence barriers around the role-dependent blocks).
    const bool interior = __all_sync(0xffffffffu, tid < NI);
    int ei = 0, ej = 0, role = 16;
    if (interior) {
        // a warp holds rows w and w + TY/2: the two 16-lane halves then fall in disjoint shared-memory banks
        role = 0;
        ei = tid & 15;
        ej = (tid >> 5) + ((tid >> 4) & 1) * (TY / 2);
    } else if (tid < NI + G::NXH) {
        const int u = tid - NI;
        role = u >= TY ? 2 : 1;
        ei = role == 2 ? PS : -1;
        ej = role == 2 ? u - TY : u;
    } else if (tid < NI + G::NXH + G::NYH) {
        const int u = tid - NI - G::NXH;
        role = u >= 16 ? 8 : 4;
        ei = u & 15;
        ej = role == 8 ? TY : -1;
    }
    const bool pub_x = (role & ~1) == 0, pub_y = (role & ~4) == 0;      // publishes x+ / y+
    const bool own_x = (role & ~2) == 0, own_y = (role & ~8) == 0;      // solves its lower x / y face
    const int gj = j0 + ej;
    MhmCell<T> c;
    c.cidx = (ej + NGH) * NP + (ei + NGH);
    c.sx_own = ej * G::SW + ei;
    c.sy_own = ej * G::SW + ei;
    c.gin_off = NGH * (NP * NP) + (gj + NGH) * NP + (ei + NGH);
    c.out_off = gj * PS + ei;
    T* gout = a.out + (size_t)g * NV * (PS * PSQ);
    T* gflux = a.flux ? a.flux + (size_t)g * 9 * NV * PSQ : nullptr;     // block-uniform
    // patch-boundary x / y faces are copied from shared memory to flux_out by the halo warps,
    // one plane late, when those warps would otherwise idle: faces i = 0, 8, 16 (x) and rows with gj = 0 mod 8 (y)
    const int hid = tid - NI;
    const int yrow0 = (8 - (j0 & 7)) & 7;      // first tile row whose lower face is a patch boundary

    if (tid == 0) {
        mbar_init(&bars[0], 1);
        mbar_init(&bars[1], 1);
        mbar_fence_init();
    }
    __syncthreads();
    if (FUSED) {      // every thread issues a few copies of each plane (cp.async groups are per thread)
        stage_plane_fused_regs<T, NV, NCP>(gin, nb, cd, PF + 0, raw);
        stage_plane_fused_regs<T, NV, NCP>(gin, nb, cd, PF + 1, raw + RS);
    } else if (tid == NI) {
        issue_plane<T, NV, TY>(gin, j0, PF + 0, raw, &bars[0]);
        if (NSTG > 1) issue_plane<T, NV, TY>(gin, j0, PF + 1, raw + RS, &bars[1]);
    }
    // prologue: all threads convert staged plane n into dst, then the freed landing stage is refilled
    auto convert_all = [&](int n, T* dst) {
        if (FUSED) {
            cp_async_wait<0>();
            __syncthreads();
            convert_plane_fused<T, NV, EXT, TY, NT>(raw + (n % NSTG) * RS, dst, ph, tid);
        } else {
            mbar_wait(&bars[n % NSTG], (n / NSTG) & 1);
            convert_plane<T, NV, EXT, TY, NT>(raw + (n % NSTG) * RS, dst, ph, tid);
        }
        __syncthreads();
        if (n + NSTG < NPL) {
            if (FUSED) stage_plane_fused_regs<T, NV, NCP>(gin, nb, cd, PF + n + NSTG, raw + (n % NSTG) * RS);
            else if (tid == NI) issue_plane<T, NV, TY>(gin, j0, PF + n + NSTG, raw + (n % NSTG) * RS, &bars[n % NSTG]);
        }
    };
    Counters cnt = {0, 0, 0, 0, 0};
    T* wn = sm + G::WN;                              // VL: primitives of U^n, padded plane p in slot p % 3
    T* f1x = sm + G::F1X;
    T* f1y = sm + G::F1Y;
    T* f1z = sm + G::F1Z;                            // faces below padded plane p in buffer p & 1
    constexpr int FZB = NV * G::NF1Z;
    if constexpr (!VLS) {
        // staged planes n = 0 .. 2R: what the predictor of plane -1 reads
        for (int n = 0; n <= 2 * R; ++n) convert_all(n, prim + n * S);
    } else {
        // half-step primitives of the cell planes -2, -1, 0 (what the predictor of plane -1 reads) from padded planes 0 .. 4
        for (int n = 0; n < 3; ++n) convert_all(n, wn + n * S);
        vl_faces<T, SOLVER, NV, G, NT>(wn, wn + S, f1x, f1y, f1z + FZB, false, ph, tid, cnt);            // z faces below plane 1
        vl_faces<T, SOLVER, NV, G, NT>(wn + S, wn + 2 * S, f1x, f1y, f1z, true, ph, tid, cnt);           // plane 1, z faces below plane 2
        __syncthreads();
        for (int m = -2; m <= 0; ++m) {
            const int pm = m + NGH;
            vl_cells<T, NV, EXT, G, NT>(wn + (pm % 3) * S, f1x, f1y, f1z + (pm & 1) * FZB, f1z + ((pm + 1) & 1) * FZB,
                                        prim + (m + 2) * S, ph, tid, cnt);
            convert_all(pm + 2, wn + ((pm + 2) % 3) * S);
            if (m < 0) {
                vl_faces<T, SOLVER, NV, G, NT>(wn + ((pm + 1) % 3) * S, wn + ((pm + 2) % 3) * S, f1x, f1y, f1z + (pm & 1) * FZB, true, ph,
                                               tid, cnt);
                __syncthreads();
            }
        }
    }

    T zplus[NV];                    // evolved conserved z+ state of the plane below (rotated for z)
    T fzl[NV];                      // z flux at kk-3/2 (natural variable order)
#pragma unroll
    for (int v = 0; v < NV; ++v) { zplus[v] = T(1); fzl[v] = T(0); }
    T smax = T(0);
    // Q[m] = ring slot (offset into prim) of staged plane kk+1+m; Q[2R+1] is the slot the next plane goes to
    int Q[RING];
#pragma unroll
    for (int m = 0; m < RING; ++m) Q[m] = m * S;

#pragma unroll 1
    for (int kk = -1; kk <= PS; ++kk) {
        const bool mid = kk >= 0 && kk < PS;
        const int par = kk & 1;
        T* st_x = sm + G::ST + par * G::BLK;
        T* st_y = st_x + NV * G::NSX;
        T* fl_x = sm + G::FL + par * G::BLK;
        T* fl_y = fl_x + NV * G::NSX;
        T xminus[NV], yminus[NV], fzn[NV];
        // ------------------------------------------------------------------ predictor of plane kk
        if (interior || (mid && role != 16)) {
            const T* Pz[2 * R + 1];
#pragma unroll
            for (int m = 0; m <= 2 * R; ++m) Pz[m] = prim + Q[m] + c.cidx;
            // Pass 0 evolves the six face states over dt/2; if one of them comes out unphysical the whole
            // predictor is redone with a zero increment (pass 1), which yields the un-evolved face values (R6).
            // A loop (not a branch that keeps everything alive) so that each conserved face state dies as soon
            // as it has been evolved; x+ / y+ go to shared memory at once, pass 1 simply overwrites them.
            T zminus[NV], znew[NV];
#pragma unroll 1
            for (int pass = VLS ? 1 : 0; pass < 2; ++pass) {      // VL: plain face values of the half-step state, nothing to evolve
                T Uf[3][2][NV], dU[NV], Ue[NV];
                mhm_face_states<T, RECON, NV, EXT, PLN>(Pz, ph, Uf, dU);
                const T hl = pass ? T(0) : ph.hlam;
                const bool fl_ok = pass == 0;
                bool ok;
                if constexpr (sizeof(T) == 4 && !EXT) {
                    T Um[NV], Up[NV];
                    ok = mhm_evolve_pair<NV>(Uf[0][0], Uf[0][1], dU, hl, Um, Up);
                    if (mid && pub_x) {
                        T rot[NV];
#pragma unroll
                        for (int k = 0; k < NV; ++k) rot[k] = Up[nat_index(0, k)];
                        put_state<T, NV>(st_x, G::NSX, c.sx_own + 1, rot);
                    }
#pragma unroll
                    for (int k = 0; k < NV; ++k) xminus[k] = Um[nat_index(0, k)];
                    ok = mhm_evolve_pair<NV>(Uf[1][0], Uf[1][1], dU, hl, Um, Up) && ok;
                    if (mid && pub_y) {
                        T rot[NV];
#pragma unroll
                        for (int k = 0; k < NV; ++k) rot[k] = Up[nat_index(1, k)];
                        put_state<T, NV>(st_y, G::NSY, c.sy_own + G::SW, rot);
                    }
#pragma unroll
                    for (int k = 0; k < NV; ++k) yminus[k] = Um[nat_index(1, k)];
                    ok = mhm_evolve_pair<NV>(Uf[2][0], Uf[2][1], dU, hl, Um, Up) && ok;
#pragma unroll
                    for (int k = 0; k < NV; ++k) { zminus[k] = Um[nat_index(2, k)]; znew[k] = Up[nat_index(2, k)]; }
                } else {
                ok = mhm_evolve<T, NV, EXT>(Uf[0][1], dU, hl, Ue, fl_ok, ph);
                if (mid && pub_x) {
                    T rot[NV];
#pragma unroll
                    for (int k = 0; k < NV; ++k) rot[k] = Ue[nat_index(0, k)];
                    put_state<T, NV>(st_x, G::NSX, c.sx_own + 1, rot);
                }
                ok = mhm_evolve<T, NV, EXT>(Uf[1][1], dU, hl, Ue, fl_ok, ph) && ok;
                if (mid && pub_y) {
                    T rot[NV];
#pragma unroll
                    for (int k = 0; k < NV; ++k) rot[k] = Ue[nat_index(1, k)];
                    put_state<T, NV>(st_y, G::NSY, c.sy_own + G::SW, rot);
                }
                ok = mhm_evolve<T, NV, EXT>(Uf[0][0], dU, hl, Ue, fl_ok, ph) && ok;
#pragma unroll
                for (int k = 0; k < NV; ++k) xminus[k] = Ue[nat_index(0, k)];
                ok = mhm_evolve<T, NV, EXT>(Uf[1][0], dU, hl, Ue, fl_ok, ph) && ok;
#pragma unroll
                for (int k = 0; k < NV; ++k) yminus[k] = Ue[nat_index(1, k)];
                ok = mhm_evolve<T, NV, EXT>(Uf[2][0], dU, hl, Ue, fl_ok, ph) && ok;
#pragma unroll
                for (int k = 0; k < NV; ++k) zminus[k] = Ue[nat_index(2, k)];
                ok = mhm_evolve<T, NV, EXT>(Uf[2][1], dU, hl, Ue, fl_ok, ph) && ok;
#pragma unroll
                for (int k = 0; k < NV; ++k) znew[k] = Ue[nat_index(2, k)];
                }
                if (ok || pass) break;
                cnt.reverted++;
            }
            if (interior) {
                // ------------------------------------------------------------ z face kk-1/2
                if (kk >= 0) {
                    T F[NV];
                    cnt.roe_fb += riemann_flux_cons<T, SOLVER, NV>(zplus, zminus, F, ph) ? 1 : 0;
#pragma unroll
                    for (int v = 0; v < NV; ++v) fzn[v] = F[rot_index(2, v)];
                    if (gflux != nullptr && (kk & 7) == 0) {      // block-uniform: a real branch
                        T* q = gflux + (2 * 3 + (kk >> 3)) * NV * PSQ + c.out_off;
#pragma unroll
                        for (int v = 0; v < NV; ++v) q[v * PSQ] = fzn[v];
                    }
                }
#pragma unroll
                for (int k = 0; k < NV; ++k) zplus[k] = znew[k];
            }
        }
        // ------------------------------------------------------------------ VL: first-order fluxes of the plane two above
        if constexpr (VLS) {
            const int pm = kk + 2 + NGH;
            if (pm <= PS + 1 + NGH)
                vl_faces<T, SOLVER, NV, G, NT>(wn + (pm % 3) * S, wn + ((pm + 1) % 3) * S, f1x, f1y, f1z + ((pm + 1) & 1) * FZB, true, ph, tid, cnt);
        }
        // ------------------------------------------------------------------ halo warps: next plane -> primitives
        {
            const int n = kk + CV;
            if (!interior && n < NPL) {
                T* dst = VLS ? wn + (n % 3) * S : prim + Q[2 * R + 1];
                if (FUSED) {      // this plane's copies were waited for before the previous barrier
                    convert_plane_fused<T, NV, EXT, TY, G::NCV>(raw + (n % NSTG) * RS, dst, ph, tid - NI);
                } else {
                    mbar_wait(&bars[n % NSTG], (n / NSTG) & 1);
                    convert_plane<T, NV, EXT, TY, G::NCV>(raw + (n % NSTG) * RS, dst, ph, tid - NI);
                }
            }
        }
        if (FUSED) cp_async_wait<0>();      // the plane issued one barrier ago: visible to the converting warps after this one
        __syncthreads();
        {      // the stage the plane above came from is free again
            const int n = kk + CV + NSTG;
            if (n < NPL) {
                if (FUSED) stage_plane_fused_regs<T, NV, NCP>(gin, nb, cd, PF + n, raw + (n % NSTG) * RS);
                else if (tid == NI) issue_plane<T, NV, TY>(gin, j0, PF + n, raw + (n % NSTG) * RS, &bars[n % NSTG]);
            }
        }
        // ------------------------------------------------------------------ conserved input of cell (ei, ej, kk-1)
        const bool upd = interior && kk >= 1;
        // padded mode: cell of the padded slab; fused mode: cell of this group's unpadded state
        const T* gcell = FUSED ? gin + (size_t)nb[13] * NV * (PS * PSQ) + c.out_off + (kk - 1) * PSQ
                               : gin + c.gin_off + (kk - 1) * (NP * NP);
        T U[NV];
        if (upd) {
#pragma unroll
            for (int v = 0; v < NV; ++v) U[v] = __ldg(gcell + (size_t)v * (FUSED ? PS * PSQ : NPC));
        }
        // ------------------------------------------------------------------ x and y faces of plane kk
        if (mid && own_x) {
            T WL[NV], F[NV], fn[NV];
            get_state<T, NV>(st_x, G::NSX, c.sx_own, WL);
            cnt.roe_fb += riemann_flux_cons<T, SOLVER, NV>(WL, xminus, F, ph) ? 1 : 0;
#pragma unroll
            for (int v = 0; v < NV; ++v) fn[v] = F[rot_index(0, v)];
            put_state<T, NV>(fl_x, G::NSX, c.sx_own, fn);
        }
        if (mid && own_y) {
            T WL[NV], F[NV], fn[NV];
            get_state<T, NV>(st_y, G::NSY, c.sy_own, WL);
            cnt.roe_fb += riemann_flux_cons<T, SOLVER, NV>(WL, yminus, F, ph) ? 1 : 0;
#pragma unroll
            for (int v = 0; v < NV; ++v) fn[v] = F[rot_index(1, v)];
            put_state<T, NV>(fl_y, G::NSY, c.sy_own, fn);
        }
        // ------------------------------------------------------------------ halo warps: boundary fluxes of plane kk-1
        if (!interior && kk >= 1 && gflux != nullptr) {
            const T* pl_x = sm + G::FL + (par ^ 1) * G::BLK;
            const T* pl_y = pl_x + NV * G::NSX;
            constexpr int NXF = 3 * TY, NYF = 3 * 16;
            for (int f = hid; f < NXF + NYF; f += G::NCV) {
                T fn[NV];
                T* q;
                if (f < NXF) {
                    const int p = f / TY, j = f - p * TY;
                    get_state<T, NV>(pl_x, G::NSX, j * G::SW + 8 * p, fn);
                    q = gflux + ((0 * 3 + p) * NV) * PSQ + (kk - 1) * PS + (j0 + j);
                } else {
                    const int h = f - NXF, r = h >> 4, i = h & 15;
                    const int j = yrow0 + 8 * r;
                    if (j > TY) continue;
                    get_state<T, NV>(pl_y, G::NSY, j * G::SW + i, fn);
                    q = gflux + ((1 * 3 + ((j0 + j) >> 3)) * NV) * PSQ + (kk - 1) * PS + i;
                }
#pragma unroll
                for (int v = 0; v < NV; ++v) q[v * PSQ] = fn[v];
            }
        }
        // ------------------------------------------------------------------ finish cell (ei, ej, kk-1)
        if (upd) {   // its four x/y fluxes were published before the barrier
            const T* pl_x = sm + G::FL + (par ^ 1) * G::BLK;
            const T* pl_y = pl_x + NV * G::NSX;
            T fl[NV], fr[NV], fd[NV], fu[NV];
            get_state<T, NV>(pl_x, G::NSX, c.sx_own, fl);
            get_state<T, NV>(pl_x, G::NSX, c.sx_own + 1, fr);
            get_state<T, NV>(pl_y, G::NSY, c.sy_own, fd);
            get_state<T, NV>(pl_y, G::NSY, c.sy_own + G::SW, fu);
#pragma unroll
            for (int v = 0; v < NV; ++v)
                U[v] = U[v] - ph.lam * (((fr[v] - fl[v]) + (fu[v] - fd[v])) + (fzn[v] - fzl[v]));
            close_cell<T, SOLVER, NV, EXT>(U, gcell, cnt, ph);
            T* o = gout + c.out_off + (kk - 1) * PSQ;
#pragma unroll
            for (int v = 0; v < NV; ++v) o[(size_t)v * (PS * PSQ)] = U[v];
            if (a.speed) {
                const T s = signal_speed<T, NV, MHM, EXT>(U, ph);
                smax = speed_max(smax, s);
            }
        }
        if (interior && kk >= 0) {
#pragma unroll
            for (int v = 0; v < NV; ++v) fzl[v] = fzn[v];
        }
        if constexpr (VLS) {      // half-step primitives of the plane two above into the spare ring slot; second barrier of the plane
            const int pm = kk + 2 + NGH;
            if (pm <= PS + 1 + NGH)
                vl_cells<T, NV, EXT, G, NT>(wn + (pm % 3) * S, f1x, f1y, f1z + (pm & 1) * FZB, f1z + ((pm + 1) & 1) * FZB,
                                            prim + Q[2 * R + 1], ph, tid, cnt);
            __syncthreads();
        }
        // rotate the ring: the slot of the lowest plane is the one the plane after next is converted into
        {
            const int q0 = Q[0];
#pragma unroll
            for (int m = 0; m + 1 < RING; ++m) Q[m] = Q[m + 1];
            Q[RING - 1] = q0;
        }
    }

    block_epilogue<T, NT, G::NTILE, EXT>(a, g, smax, cnt, sm, tid);
}

}  // namespace gamer
