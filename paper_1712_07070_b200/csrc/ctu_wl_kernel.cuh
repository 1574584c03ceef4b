// ctu_wl_kernel.cuh -- the WORK-LIST form of the CTU kernel, used for fp64 only.
//
// The thread-owned form (ctu_kernel.cuh) keeps a cell's six traced states, its first-pass and final fluxes in registers;
// in fp64 that is more than the 255 registers a thread can have and the tile that still fits leaves 6 warps per SM
// (measured 1.40e9 cells/s against 1.94e9 for this kernel, CTU+PPM+HLLC, 32,768 groups).  Here every stage is a flat list
// of work items (cells x directions, faces) spread over all threads and everything is exchanged through shared memory:
//
// Iteration kk = -1..17 works on three planes at once (4 block barriers per iteration):
//   T    (kk)   : PLM/PPM face values + characteristic tracing over dt/2 of every cell of plane kk
//                 (18 x (TY+2) cells, three directions)                         -> ts[kk&1]
//   R1z  (kk)   : first-pass z flux H* at kk-1/2 from ts[(kk-1)&1].z+ and ts[kk&1].z-  -> f1z[kk&1]
//                 (meanwhile the next staged plane is converted to primitives)
//   C    (kk-1) : transverse flux-gradient correction (coefficient dt/2dh, conserved variables) of
//                 the face states of plane kk-1, in place, using F*x,G*y of plane kk-1 and H* at
//                 kk-3/2, kk-1/2; corrected z+ also saved to zp[(kk-1)&1]
//   R1xy (kk)   : first-pass F*x, G*y of plane kk (overwrite those of kk-1, now consumed)
//   R2   (kk-1) : final Riemann pass of plane kk-1 (x, y faces; z faces at kk-3/2)  -> fx/fy/fz, flux_out
//   U    (kk-2) : conservative update + closing step of plane kk-2 (thread-owned cell, registers)
#pragma once
#include "hydro_close.cuh"

namespace gamer {

template <typename T, int RECON, int NV, int TY, bool FUSED = false> struct CtuWlSmem {
    using G = Geo<TY>;
    static constexpr int R = RECON == PPM ? 2 : 1;
    static constexpr int PR = 2 * R + 1;
    // every face-state / flux array is [Vec4 n | (NV-4) scalars n] in the rotated order of its axis
    // (rho, v_d, v_d+1, v_d+2, P [, q]); n is rounded up to a multiple of 4 to keep the Vec4 parts 16-byte aligned
    static constexpr int pad4(int n) { return (n + 3) / 4 * 4; }
    static constexpr int NF1X = 17 * G::EH, NF1Y = 18 * (G::EH - 1);
    static constexpr int NF1XP = pad4(NF1X), NF1YP = pad4(NF1Y);
    static constexpr int RAW = 0;                                   // [2][NV][PLN]
    static constexpr int RSTG = NV * (FUSED ? G::NR * FW : G::PLN); // one landing stage (fused refresh: 24-wide rows)
    static constexpr int PRIM = RAW + 2 * RSTG;                     // [PR][NV][PLN]
    static constexpr int TS = PRIM + PR * NV * G::PLN;              // [2][6] x state array of EPL
    static constexpr int F1X = TS + 2 * 6 * NV * G::EPL;            // flux array of NF1XP
    static constexpr int F1Y = F1X + NV * NF1XP;                    // flux array of NF1YP
    static constexpr int F1Z = F1Y + NV * NF1YP;                    // [2] x flux array of EPL
    static constexpr int ZP = F1Z + 2 * NV * G::EPL;                // [2] x state array of NFZ
    static constexpr int FX = ZP + 2 * NV * G::NFZ;
    static constexpr int FY = FX + NV * G::NFX;
    static constexpr int FZ = FY + NV * G::NFY;
    static constexpr int END = FZ + NV * G::NFZ;
    static_assert(RSTG % 4 == 0 && (NV * G::PLN) % 4 == 0 && G::EPL % 4 == 0 && G::NFX % 4 == 0 && G::NFY % 4 == 0 && G::NFZ % 4 == 0,
                  "16-byte alignment of the Vec4 arrays");
    static constexpr size_t BYTES = 16 + (size_t)END * sizeof(T) + (FUSED ? 128 : 0);   // + neighbour table
};

// one first-pass Riemann solve: states and flux are stored in the rotated order of the axis, nothing to rotate here
template <typename T, int SOLVER, int NV>
__device__ __forceinline__ int first_pass_face(const T* lblk, int lidx, const T* rblk, int ridx, int sn, T* fblk,
                                               int fidx, int fn, const Phys<T>& ph) {
    T WL[NV], WR[NV], F[NV];
    get_state<T, NV>(lblk, sn, lidx, WL);
    get_state<T, NV>(rblk, sn, ridx, WR);
    const int fb = riemann_flux<T, SOLVER, NV>(WL, WR, F, ph) ? 1 : 0;
    put_state<T, NV>(fblk, fn, fidx, F);
    return fb;
}

// final Riemann pass over the faces of one plane of the tile (x- and y-faces of plane kk, z-faces between planes kk-1 and
// kk): es = the six corrected state arrays of the plane, zprev = corrected z+ of plane kk-1; fluxes go to fx/fy/fz in the
// rotated order of their axis and, on patch boundaries, to flux_out in natural order
template <typename T, int SOLVER, int NV, int TY, int NT>
__device__ __forceinline__ int ctu_final_pass(const T* es, const T* zprev, T* fx, T* fy, T* fz, T* gflux, int kk, int j0,
                                              const Phys<T>& ph, int tid) {
    using G = Geo<TY>;
    constexpr int SB = NV * G::EPL;      // one state array
    int nfb = 0;
    const int f_lo = (kk >= 0 && kk < PS) ? 0 : G::NFX + G::NFY;
    const int f_hi = (kk >= 0 && kk <= PS) ? G::NF : 0;
    for (int f = f_lo + tid; f < f_hi; f += NT) {
        int d, lidx, ridx, ln, fidx, fn, gp, ga, gb;
        const T *lp, *rp;
        T* fp;
        if (f < G::NFX) {
            const int jj = f / 17, ii = f - jj * 17;
            d = 0;
            lp = es + 1 * SB; lidx = (jj + 1) * G::EW + ii; ln = G::EPL;
            rp = es + 0 * SB; ridx = lidx + 1;
            fp = fx; fidx = f; fn = G::NFX;
            gp = ii; ga = j0 + jj; gb = kk;
        } else if (f < G::NFX + G::NFY) {
            const int g = f - G::NFX;
            const int jj = g >> 4, ii = g & 15;
            d = 1;
            lp = es + 3 * SB; lidx = jj * G::EW + ii + 1; ln = G::EPL;
            rp = es + 2 * SB; ridx = lidx + G::EW;
            fp = fy; fidx = g; fn = G::NFY;
            gp = j0 + jj; ga = ii; gb = kk;
        } else {
            const int g = f - G::NFX - G::NFY;
            const int jj = g >> 4, ii = g & 15;
            d = 2;
            lp = zprev; lidx = g; ln = G::NFZ;
            rp = es + 4 * SB; ridx = (jj + 1) * G::EW + ii + 1;
            fp = fz; fidx = g; fn = G::NFZ;
            gp = kk; ga = ii; gb = j0 + jj;
        }
        T WL[NV], WR[NV], F[NV];
        get_state<T, NV>(lp, ln, lidx, WL);
        get_state<T, NV>(rp, G::EPL, ridx, WR);
        nfb += riemann_flux<T, SOLVER, NV>(WL, WR, F, ph) ? 1 : 0;
        put_state<T, NV>(fp, fn, fidx, F);
        if (gflux != nullptr && (gp & 7) == 0) {   // faces 0, 8, 16 of the axis: patch boundaries (L112)
            const int cn = 1 + d, c1 = 1 + (d + 1) % 3, c2 = 1 + (d + 2) % 3;
            T* q = gflux + ((size_t)(d * 3 + (gp >> 3)) * NV) * (PS * PS) + gb * PS + ga;
            q[0] = F[0];
            q[(size_t)cn * (PS * PS)] = F[1];
            q[(size_t)c1 * (PS * PS)] = F[2];
            q[(size_t)c2 * (PS * PS)] = F[3];
            q[(size_t)4 * (PS * PS)] = F[4];
#pragma unroll
            for (int v = 5; v < NV; ++v) q[(size_t)v * (PS * PS)] = F[v];
        }
    }
    return nfb;
}

// One work list for the two Riemann passes that share a phase: the first-pass x / y faces of plane kk (states tcur ->
// f1x, f1y) followed by the final-pass faces of plane m = kk-1 (corrected states tprev, zprev -> fx, fy, fz and flux_out).
// A single list keeps all threads busy for ceil(total / NT) rounds instead of ceil(n1 / NT) + ceil(n2 / NT), and a single
// call site keeps one copy of the solver in the instruction stream.
template <typename T, int RECON, int SOLVER, int NV, int TY, int NT, bool FUSED>
__device__ __forceinline__ int ctu_riemann_phase(const T* tcur, const T* tprev, const T* zprev, T* f1x, T* f1y, T* fx, T* fy,
                                                 T* fz, T* gflux, int kk, int j0, const Phys<T>& ph, int tid) {
    using G = Geo<TY>;
    using S = CtuWlSmem<T, RECON, NV, TY, FUSED>;
    constexpr int SB = NV * G::EPL, EW = G::EW;
    const int m = kk - 1;
    const int n1 = kk <= PS ? S::NF1X + S::NF1Y : 0;
    const int f_lo = (m >= 0 && m < PS) ? 0 : G::NFX + G::NFY;
    const int f_hi = (m >= 0 && m <= PS) ? G::NF : f_lo;
    int nfb = 0;
    for (int it = tid; it < n1 + (f_hi - f_lo); it += NT) {
        int d, lidx, ridx, ln, fidx, fn, gp = 1, ga = 0, gb = 0;
        const T *lp, *rp;
        T* fp;
        if (it < S::NF1X && it < n1) {                      // first pass, x face of plane kk
            const int ej = it / 17, ei = it - ej * 17;
            d = 0;
            lp = tcur + 1 * SB; lidx = ej * EW + ei; ln = G::EPL;
            rp = tcur + 0 * SB; ridx = lidx + 1;
            fp = f1x; fidx = it; fn = S::NF1XP;
        } else if (it < n1) {                               // first pass, y face
            const int u = it - S::NF1X;
            d = 1;
            lp = tcur + 3 * SB; lidx = u; ln = G::EPL;
            rp = tcur + 2 * SB; ridx = u + EW;
            fp = f1y; fidx = u; fn = S::NF1YP;
        } else {                                            // final pass of plane m
            const int f = it - n1 + f_lo;
            if (f < G::NFX) {
                const int jj = f / 17, ii = f - jj * 17;
                d = 0;
                lp = tprev + 1 * SB; lidx = (jj + 1) * EW + ii; ln = G::EPL;
                rp = tprev + 0 * SB; ridx = lidx + 1;
                fp = fx; fidx = f; fn = G::NFX;
                gp = ii; ga = j0 + jj; gb = m;
            } else if (f < G::NFX + G::NFY) {
                const int g = f - G::NFX;
                const int jj = g >> 4, ii = g & 15;
                d = 1;
                lp = tprev + 3 * SB; lidx = jj * EW + ii + 1; ln = G::EPL;
                rp = tprev + 2 * SB; ridx = lidx + EW;
                fp = fy; fidx = g; fn = G::NFY;
                gp = j0 + jj; ga = ii; gb = m;
            } else {
                const int g = f - G::NFX - G::NFY;
                const int jj = g >> 4, ii = g & 15;
                d = 2;
                lp = zprev; lidx = g; ln = G::NFZ;
                rp = tprev + 4 * SB; ridx = (jj + 1) * EW + ii + 1;
                fp = fz; fidx = g; fn = G::NFZ;
                gp = m; ga = ii; gb = j0 + jj;
            }
        }
        T WL[NV], WR[NV], F[NV];
        get_state<T, NV>(lp, ln, lidx, WL);
        get_state<T, NV>(rp, G::EPL, ridx, WR);
        nfb += riemann_flux<T, SOLVER, NV>(WL, WR, F, ph) ? 1 : 0;
        put_state<T, NV>(fp, fn, fidx, F);
        if (gflux != nullptr && it >= n1 && (gp & 7) == 0) {   // final pass on faces 0, 8, 16: patch boundaries (L112)
            const int cn = 1 + d, c1 = 1 + (d + 1) % 3, c2 = 1 + (d + 2) % 3;
            T* q = gflux + ((size_t)(d * 3 + (gp >> 3)) * NV) * (PS * PS) + gb * PS + ga;
            q[0] = F[0];
            q[(size_t)cn * (PS * PS)] = F[1];
            q[(size_t)c1 * (PS * PS)] = F[2];
            q[(size_t)c2 * (PS * PS)] = F[3];
            q[(size_t)4 * (PS * PS)] = F[4];
#pragma unroll
            for (int v = 5; v < NV; ++v) q[(size_t)v * (PS * PS)] = F[v];
        }
    }
    return nfb;
}

// T stage for one cell t of the 18 x (TY+2) face-state plane and one direction D: PLM/PPM face values of
// every variable along D, characteristic tracing over dt/2 (R7), revert of an unphysical pair (R8), store.
template <typename T, int RECON, int NV, bool EXT, int TY, int D>
__device__ __forceinline__ void ctu_trace_dir(const T* const* Pz, int t, T* tcur, const Phys<T>& ph, Counters& cnt) {
    using G = Geo<TY>;
    constexpr int R = RECON == PPM ? 2 : 1;
    constexpr int EPL = G::EPL, EW = G::EW;
    constexpr int cn = 1 + D, c1 = 1 + (D + 1) % 3, c2 = 1 + (D + 2) % 3;
    const int ej = t / EW, ei = t - ej * EW;
    const int c = (ej + 2) * NP + (ei + 2);
    T Wr[NV], rm[NV], rp[NV], tm[NV], tp[NV];
    if (EXT && ph.char_limit) {      // slopes limited in characteristic variables (R22): all variables together
        T W5[5][NV];
#pragma unroll
        for (int m = -R; m <= R; ++m) {
            const T* q = (D == 2) ? Pz[R + m] + c : Pz[R] + c + m * (D == 0 ? 1 : NP);
            W5[m + 2][0] = q[0]; W5[m + 2][1] = q[cn * G::PLN]; W5[m + 2][2] = q[c1 * G::PLN]; W5[m + 2][3] = q[c2 * G::PLN];
            W5[m + 2][4] = q[4 * G::PLN];
#pragma unroll
            for (int v = 5; v < NV; ++v) W5[m + 2][v] = q[v * G::PLN];
        }
#pragma unroll
        for (int k = 0; k < NV; ++k) Wr[k] = W5[2][k];
        face_values_char<T, RECON, NV, EXT>(W5, rm, rp, ph);
    } else {
        T wm[NV], wp[NV], Wc[NV];
#pragma unroll
        for (int v = 0; v < NV; ++v) {
            const T* q = Pz[R] + v * G::PLN + c;
            Wc[v] = q[0];
            if (D == 0) face_values<T, RECON, EXT, fixed_theta(EXT, RECON)>(q, 1, wm[v], wp[v], ph);
            else if (D == 1) face_values<T, RECON, EXT, fixed_theta(EXT, RECON)>(q, NP, wm[v], wp[v], ph);
            else {
                const int o = v * G::PLN + c;
                if (RECON == PPM)
                    face_values5<T, RECON, EXT>(Pz[0][o], Pz[R - 1][o], Pz[R][o], Pz[R + 1][o], Pz[2 * R][o], wm[v], wp[v], ph);
                else
                    face_values5<T, RECON, EXT>(T(0), Pz[R - 1][o], Pz[R][o], Pz[R + 1][o], T(0), wm[v], wp[v], ph);
            }
        }
        // rotate so that the traced axis is "n"
        Wr[0] = Wc[0]; Wr[1] = Wc[cn]; Wr[2] = Wc[c1]; Wr[3] = Wc[c2]; Wr[4] = Wc[4];
        rm[0] = wm[0]; rm[1] = wm[cn]; rm[2] = wm[c1]; rm[3] = wm[c2]; rm[4] = wm[4];
        rp[0] = wp[0]; rp[1] = wp[cn]; rp[2] = wp[c1]; rp[3] = wp[c2]; rp[4] = wp[4];
#pragma unroll
        for (int v = 5; v < NV; ++v) { Wr[v] = Wc[v]; rm[v] = wm[v]; rp[v] = wp[v]; }
    }
    trace_cell<T, RECON, NV>(Wr, rm, rp, tm, tp, ph);
    if (EXT && ph.floors) { floor_prim(tm, ph); floor_prim(tp, ph); }
    if (!(tm[0] > T(0) && tm[4] > T(0) && tp[0] > T(0) && tp[4] > T(0))) {
        cnt.reverted++;
#pragma unroll
        for (int v = 0; v < NV; ++v) { tm[v] = rm[v]; tp[v] = rp[v]; }
    }
    put_state<T, NV>(tcur + (2 * D) * NV * EPL, EPL, t, tm);          // rotated for axis D, as traced
    put_state<T, NV>(tcur + (2 * D + 1) * NV * EPL, EPL, t, tp);
}

template <typename T, int RECON, int SOLVER, int NV, bool EXT, int TY, int NT, bool FUSED>
__global__ void __launch_bounds__(NT) ctu_wl_kernel(const AdvArgs<T> a) {
    using G = Geo<TY>;
    using S = CtuWlSmem<T, RECON, NV, TY, FUSED>;
    constexpr int RS = S::RSTG;
    constexpr int R = S::R, PR = S::PR;
    constexpr int NPL = 18 + 2 * R;
    constexpr int PF = 2 - R;
    constexpr int EPL = G::EPL, EW = G::EW;

    extern __shared__ __align__(128) unsigned char smem_raw[];
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem_raw);
    T* sm = reinterpret_cast<T*>(smem_raw + 16);
    T* raw = sm + S::RAW;
    T* prim = sm + S::PRIM;
    T* ts = sm + S::TS;
    T* f1x = sm + S::F1X;
    T* f1y = sm + S::F1Y;
    T* f1z = sm + S::F1Z;
    T* zp = sm + S::ZP;
    T* fx = sm + S::FX;
    T* fy = sm + S::FY;
    T* fz = sm + S::FZ;

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
    T* gout = a.out + (size_t)g * NV * (PS * PS * PS);
    T* gflux = a.flux ? a.flux + (size_t)g * 9 * NV * (PS * PS) : nullptr;
    const Phys<T> ph = make_phys<T>(a);

    if (tid == 0) {
        mbar_init(&bars[0], 1);
        mbar_init(&bars[1], 1);
        mbar_fence_init();
    }
    __syncthreads();
    if (FUSED) {
        stage_plane_fused_regs<T, NV, NCD>(gin, nb, cd, PF + 0, raw);
        stage_plane_fused_regs<T, NV, NCD>(gin, nb, cd, PF + 1, raw + RS);
    } else if (tid == 0) {
        issue_plane<T, NV, TY>(gin, j0, PF + 0, raw, &bars[0]);
        issue_plane<T, NV, TY>(gin, j0, PF + 1, raw + RS, &bars[1]);
    }
    for (int n = 0; n <= 2 * R; ++n) {
        if (FUSED) {
            cp_async_wait<0>();
            __syncthreads();
            convert_plane_fused<T, NV, EXT, TY, NT>(raw + (n & 1) * RS, prim + ((PF + n) % PR) * NV * G::PLN, ph, tid);
        } else {
            mbar_wait(&bars[n & 1], (n >> 1) & 1);
            convert_plane<T, NV, EXT, TY, NT>(raw + (n & 1) * RS, prim + ((PF + n) % PR) * NV * G::PLN, ph, tid);
        }
        __syncthreads();
        if (n + 2 < NPL) {
            if (FUSED) stage_plane_fused_regs<T, NV, NCD>(gin, nb, cd, PF + n + 2, raw + (n & 1) * RS);
            else if (tid == 0) issue_plane<T, NV, TY>(gin, j0, PF + n + 2, raw + (n & 1) * RS, &bars[n & 1]);
        }
    }

    const bool owner = tid < G::NFZ;           // threads that own a cell column of the update
    const int ci = tid & 15, cj = (tid >> 4) % TY;
    T sxy[NV], fzm[NV];
#pragma unroll
    for (int v = 0; v < NV; ++v) { sxy[v] = T(0); fzm[v] = T(0); }
    T smax = T(0);
    Counters cnt = {0, 0, 0, 0, 0};

    for (int kk = -1; kk <= PS + 1; ++kk) {
        T* tcur = ts + (kk & 1) * 6 * NV * EPL;            // plane kk
        T* tprev = ts + ((kk + 1) & 1) * 6 * NV * EPL;     // plane kk-1
        const int m = kk - 1;
        // ------------------------------------------------------------------ T(kk)
        // work item = (direction, cell): 3 * EPL items spread over all NT threads
        if (kk <= PS) {
            const int pc = kk + NGH;
            const T* Pz[2 * R + 1];
#pragma unroll
            for (int q = -R; q <= R; ++q) Pz[q + R] = prim + ((pc + q) % PR) * NV * G::PLN;
            for (int item = tid; item < 3 * EPL; item += NT) {
                const int d = item / EPL, t = item - d * EPL;
                if (d == 0) ctu_trace_dir<T, RECON, NV, EXT, TY, 0>(Pz, t, tcur, ph, cnt);
                else if (d == 1) ctu_trace_dir<T, RECON, NV, EXT, TY, 1>(Pz, t, tcur, ph, cnt);
                else ctu_trace_dir<T, RECON, NV, EXT, TY, 2>(Pz, t, tcur, ph, cnt);
            }
        }
        if (FUSED) cp_async_wait<0>();      // this thread's share of the plane converted below
        __syncthreads();
        // ------------------------------------------------------------------ R1z(kk) + convert
        if (kk >= 0 && kk <= PS) {
            T* hz = f1z + (kk & 1) * NV * EPL;
            for (int t = tid; t < EPL; t += NT)
                cnt.roe_fb += first_pass_face<T, SOLVER, NV>(tprev + 5 * NV * EPL, t, tcur + 4 * NV * EPL, t, EPL, hz, t, EPL, ph);
        }
        {
            const int n = kk + 2 + 2 * R;
            if (n < NPL) {
                if (FUSED) {      // copies waited for before the barrier above
                    convert_plane_fused<T, NV, EXT, TY, NT>(raw + (n & 1) * RS, prim + ((PF + n) % PR) * NV * G::PLN, ph, tid);
                } else {
                    mbar_wait(&bars[n & 1], (n >> 1) & 1);
                    convert_plane<T, NV, EXT, TY, NT>(raw + (n & 1) * RS, prim + ((PF + n) % PR) * NV * G::PLN, ph, tid);
                }
            }
        }
        __syncthreads();
        // ------------------------------------------------------------------ C(kk-1)
        if (m >= -1 && m <= PS) {
            const bool mid = (m >= 0 && m < PS);            // x/y states are needed only in planes 0..15
            const T* hlo = f1z + (m & 1) * NV * EPL;        // H* at m-1/2
            const T* hhi = f1z + (kk & 1) * NV * EPL;       // H* at m+1/2
            T* zsave = zp + (m & 1) * NV * G::NFZ;
            for (int t = tid; t < G::NPLUS; t += NT) {
                int ei, ej;
                if (t < 18 * TY) { ej = t / 18; ei = t - ej * 18; ej += 1; }
                else { const int u = t - 18 * TY; ej = (u < 16) ? 0 : TY + 1; ei = 1 + (u & 15); }
                const int e = ej * EW + ei;
                const bool rowin = (ej >= 1 && ej <= TY), colin = (ei >= 1 && ei <= 16);
                T gx[NV], gy[NV], gz[NV];     // flux differences across the cell in x, y, z (natural variable order)
#pragma unroll
                for (int v = 0; v < NV; ++v) gx[v] = gy[v] = gz[v] = T(0);
                if (colin) {
                    T A[NV], B[NV];
                    get_state<T, NV>(f1x, S::NF1XP, ej * 17 + ei, A);
                    get_state<T, NV>(f1x, S::NF1XP, ej * 17 + ei - 1, B);
#pragma unroll
                    for (int k = 0; k < NV; ++k) gx[nat_index(0, k)] = A[k] - B[k];
                }
                if (rowin) {
                    T A[NV], B[NV];
                    get_state<T, NV>(f1y, S::NF1YP, ej * 18 + ei, A);
                    get_state<T, NV>(f1y, S::NF1YP, (ej - 1) * 18 + ei, B);
#pragma unroll
                    for (int k = 0; k < NV; ++k) gy[nat_index(1, k)] = A[k] - B[k];
                }
                if (mid) {
                    T A[NV], B[NV];
                    get_state<T, NV>(hhi, EPL, e, A);
                    get_state<T, NV>(hlo, EPL, e, B);
#pragma unroll
                    for (int k = 0; k < NV; ++k) gz[nat_index(2, k)] = A[k] - B[k];
                }
#pragma unroll
                for (int d = 0; d < 3; ++d) {
                    const bool need = (d == 0) ? (rowin && mid) : (d == 1) ? (colin && mid) : (rowin && colin);
                    if (!need) continue;
                    const T* g1 = (d == 0) ? gy : (d == 1) ? gz : gx;     // d1 = (d+1)%3
                    const T* g2 = (d == 0) ? gz : (d == 1) ? gx : gy;     // d2 = (d+2)%3
#pragma unroll
                    for (int s = 0; s < 2; ++s) {
                        T* sblk = tprev + (2 * d + s) * NV * EPL;
                        T W[NV], U[NV], Wn[NV], Wrot[NV];
                        get_state<T, NV>(sblk, EPL, e, Wrot);
#pragma unroll
                        for (int k = 0; k < NV; ++k) W[nat_index(d, k)] = Wrot[k];
                        prim2cons<T, NV>(W, U, ph);
#pragma unroll
                        for (int v = 0; v < NV; ++v) U[v] = U[v] - ph.hlam * g1[v] - ph.hlam * g2[v];
                        cons2prim<T, NV>(U, Wn, ph);
                        if (EXT && ph.floors) floor_prim(Wn, ph);
                        const bool ok = Wn[0] > T(0) && Wn[4] > T(0);
                        if (!ok) cnt.reverted++;
#pragma unroll
                        for (int k = 0; k < NV; ++k) Wrot[k] = ok ? Wn[nat_index(d, k)] : W[nat_index(d, k)];
                        if (d == 2 && s == 1) put_state<T, NV>(zsave, G::NFZ, (ej - 1) * 16 + (ei - 1), Wrot);
                        else put_state<T, NV>(sblk, EPL, e, Wrot);
                    }
                }
            }
        }
        __syncthreads();
        // ------------------------------------------------------------------ R1xy(kk) + R2(kk-1)
        if constexpr (sizeof(T) == 8) {
            // fp64 (fewer threads per CTA): one work list for both passes, see ctu_riemann_phase (+8 %; -1 % in fp32)
            cnt.roe_fb += ctu_riemann_phase<T, RECON, SOLVER, NV, TY, NT, FUSED>(tcur, tprev, zp + ((m + 1) & 1) * NV * G::NFZ, f1x,
                                                                               f1y, fx, fy, fz, gflux, kk, j0, ph, tid);
        } else {
            if (kk <= PS) {
                for (int t = tid; t < S::NF1X + S::NF1Y; t += NT) {      // one call site for x and y faces
                    const bool isx = t < S::NF1X;
                    const int u = isx ? t : t - S::NF1X;              // x: ej*17 + ei;  y: ej*18 + ei, ej in [0, EH-1)
                    const int ej = u / 17, ei = u - ej * 17;
                    const int l = isx ? ej * EW + ei : u;
                    cnt.roe_fb += first_pass_face<T, SOLVER, NV>(tcur + (isx ? 1 : 3) * NV * EPL, l, tcur + (isx ? 0 : 2) * NV * EPL,
                                                                 isx ? l + 1 : l + EW, EPL, isx ? f1x : f1y, u,
                                                                 isx ? S::NF1XP : S::NF1YP, ph);
                }
            }
            if (m >= 0) cnt.roe_fb += ctu_final_pass<T, SOLVER, NV, TY, NT>(tprev, zp + ((m + 1) & 1) * NV * G::NFZ, fx, fy, fz, gflux, m, j0, ph, tid);
        }
        __syncthreads();
        // ------------------------------------------------------------------ U(kk-2)
        {
            const int n = kk + 4 + 2 * R;
            if (n < NPL) {
                if (FUSED) stage_plane_fused_regs<T, NV, NCD>(gin, nb, cd, PF + n, raw + (n & 1) * RS);
                else if (tid == 0) issue_plane<T, NV, TY>(gin, j0, PF + n, raw + (n & 1) * RS, &bars[n & 1]);
            }
        }
        if (owner) {
            if (m >= 1) {
                const int k = m - 1;
                const T* gcell = FUSED ? gin + (size_t)nb[13] * NV * (PS * PS * PS) + (size_t)k * (PS * PS) + (j0 + cj) * PS + ci
                                       : gin + (size_t)(k + NGH) * (NP * NP) + (j0 + cj + NGH) * NP + (ci + NGH);
                T U[NV], Fz[NV];
                get_state<T, NV>(fz, G::NFZ, tid, Fz);
#pragma unroll
                for (int v = 0; v < NV; ++v) {
                    const T dfz = Fz[rot_index(2, v)] - fzm[v];
                    U[v] = __ldg(gcell + (size_t)v * (FUSED ? PS * PS * PS : NPC)) - ph.lam * (sxy[v] + dfz);
                }
                close_cell<T, SOLVER, NV, EXT>(U, gcell, cnt, ph);
#pragma unroll
                for (int v = 0; v < NV; ++v) gout[((size_t)v * PS + k) * (PS * PS) + (j0 + cj) * PS + ci] = U[v];
                if (a.speed) {
                    const T s = signal_speed<T, NV, CTU, EXT>(U, ph);
                    smax = speed_max(smax, s);
                }
            }
            if (m >= 0 && m < PS) {
                T Xr[NV], Xl[NV], Yu[NV], Yd[NV], Fz[NV];
                get_state<T, NV>(fx, G::NFX, cj * 17 + ci + 1, Xr);
                get_state<T, NV>(fx, G::NFX, cj * 17 + ci, Xl);
                get_state<T, NV>(fy, G::NFY, (cj + 1) * 16 + ci, Yu);
                get_state<T, NV>(fy, G::NFY, cj * 16 + ci, Yd);
                get_state<T, NV>(fz, G::NFZ, tid, Fz);
#pragma unroll
                for (int v = 0; v < NV; ++v) {
                    const T dfx = Xr[rot_index(0, v)] - Xl[rot_index(0, v)];
                    const T dfy = Yu[rot_index(1, v)] - Yd[rot_index(1, v)];
                    sxy[v] = dfx + dfy;
                    fzm[v] = Fz[rot_index(2, v)];
                }
            }
        }
    }

    block_epilogue<T, NT, G::NTILE, EXT>(a, g, smax, cnt, sm, tid);
}

}  // namespace gamer
