// mhm_kernel.cuh -- MUSCL-Hancock (MHM; Toro 2009 sect. 14.4/16.5) patch-group kernel.
//
// Per plane kk = -1..16 of the tile (2 block barriers per plane):
//   S1  predictor : PLM/PPM face values of the "plus"-shaped cell set of the plane (the cells whose
//                   face states a final flux needs), Hancock half-step with the cell's own face
//                   fluxes in all three directions, conversion back to primitives -> es / zp (smem)
//   S2  Riemann   : x/y faces of plane kk, z faces between kk-1 and kk -> fx/fy/fz (smem) and the
//                   patch-boundary planes of flux_out;  meanwhile the next staged plane -> primitives
//   S3  update    : thread (i,j) finishes cell (i,j,kk-1) (needs F_z at kk-1/2), applies the closing
//                   step, writes `out`, tracks the CFL maximum; then keeps (dFx+dFy) and F_z(kk-1/2)
//                   of plane kk in registers;  one thread re-arms the freed TMA stage.
#pragma once
#include "hydro_close.cuh"

namespace gamer {

template <typename T, int RECON, int NV, int TY> struct MhmSmem {
    using G = Geo<TY>;
    static constexpr int R = RECON == PPM ? 2 : 1;
    static constexpr int PR = 2 * R + 1;
    static constexpr int RAW = 0;                                   // [2][NV][PLN]
    static constexpr int PRIM = RAW + 2 * NV * G::PLN;              // [PR][NV][PLN]
    static constexpr int ES = PRIM + PR * NV * G::PLN;              // [5][NV][EPL]
    static constexpr int ZP = ES + 5 * NV * G::EPL;                 // [2][NV][EPL]  z+ of planes kk, kk-1
    static constexpr int FL = ZP + 2 * NV * G::EPL;                 // [NV][NF]      rotated fluxes, flat face list
    static constexpr int END = FL + NV * G::NF;
    static constexpr size_t BYTES = 16 + (size_t)END * sizeof(T);  // 2 mbarriers first
};

template <typename T, int RECON, int SOLVER, int NV, bool EXT, int TY, int NT, int MINB>
__global__ void __launch_bounds__(NT, MINB) mhm_kernel(const AdvArgs<T> a) {
    using G = Geo<TY>;
    using S = MhmSmem<T, RECON, NV, TY>;
    constexpr int R = S::R, PR = S::PR;
    constexpr int NPL = 18 + 2 * R;      // staged planes: padded 2-R .. 19+R
    constexpr int PF = 2 - R;

    extern __shared__ __align__(128) unsigned char smem_raw[];
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem_raw);
    T* sm = reinterpret_cast<T*>(smem_raw + 16);
    T* raw = sm + S::RAW;
    T* prim = sm + S::PRIM;
    T* es = sm + S::ES;
    T* fl = sm + S::FL;

    const int tid = threadIdx.x;
    const long long tile = blockIdx.x;
    const long long g = tile / G::NTILE;
    const int j0 = (int)(tile % G::NTILE) * TY;
    const T* gin = a.in + (size_t)g * NV * NPC;
    T* gout = a.out + (size_t)g * NV * (PS * PS * PS);
    T* gflux = a.flux ? a.flux + (size_t)g * 9 * NV * (PS * PS) : nullptr;
    const Phys<T> ph = make_phys<T>(a);

    if (tid == 0) {
        mbar_init(&bars[0], 1);
        mbar_init(&bars[1], 1);
        mbar_fence_init();
    }
    __syncthreads();
    if (tid == 0) {
        issue_plane<T, NV, TY>(gin, j0, PF + 0, raw, &bars[0]);
        issue_plane<T, NV, TY>(gin, j0, PF + 1, raw + NV * G::PLN, &bars[1]);
    }
    // prologue: fill the primitive ring with staged planes n = 0 .. 2R
    for (int n = 0; n <= 2 * R; ++n) {
        mbar_wait(&bars[n & 1], (n >> 1) & 1);
        convert_plane<T, NV, EXT, TY, NT>(raw + (n & 1) * NV * G::PLN, prim + ((PF + n) % PR) * NV * G::PLN, ph, tid);
        __syncthreads();
        if (tid == 0 && n + 2 < NPL) issue_plane<T, NV, TY>(gin, j0, PF + n + 2, raw + (n & 1) * NV * G::PLN, &bars[n & 1]);
    }

    // per-thread cell of the update stage
    const bool owner = tid < G::NFZ;               // threads that own a cell column of the update stage
    const int ci = tid & 15, cj = (tid >> 4) % TY;
    // the convert stage starts at the warps that get fewer Riemann faces, to balance the barrier interval
    constexpr int CROT = (G::NF % NT) == 0 ? 0 : ((G::NF % NT + 31) / 32) * 32 % NT;
    const int ctid = (tid + NT - CROT) % NT;
    // loop-invariant face descriptors of this thread's Riemann rounds (f = tid + r*NT)
    constexpr int NROUND = (G::NF + NT - 1) / NT;
    constexpr int ZOFF = 5 * NV * G::EPL;          // offset of the z+ buffers relative to es
    unsigned fdesc[NROUND];
#pragma unroll
    for (int r = 0; r < NROUND; ++r) fdesc[r] = face_descriptor<NV, TY>(tid + r * NT < G::NF ? tid + r * NT : 0, ZOFF);
    T sxy[NV], fzm[NV];
#pragma unroll
    for (int v = 0; v < NV; ++v) { sxy[v] = T(0); fzm[v] = T(0); }
    T smax = T(0);
    Counters cnt = {0, 0, 0, 0, 0};

    int slot0 = (NGH - 1 - R) % PR;      // ring slot of the lowest plane the predictor of plane kk reads
    for (int kk = -1; kk <= PS; ++kk, slot0 = (slot0 + 1 == PR) ? 0 : slot0 + 1) {
        // ------------------------------------------------------------------ S1: predictor
        {
            const int pc = kk + NGH;   // padded plane index of kk
            const T* Pz[2 * R + 1];
#pragma unroll
            for (int m = 0; m <= 2 * R; ++m) {
                int sl = slot0 + m;
                if (sl >= PR) sl -= PR;
                Pz[m] = prim + sl * NV * G::PLN;
            }
            (void)pc;
            T* zcur = es + ZOFF + (kk & 1) * NV * G::EPL;
            for (int t = tid; t < G::NPLUS; t += NT) {
                int ei, ej;
                if (t < 18 * TY) { ej = t / 18; ei = t - ej * 18; ej += 1; }
                else { const int u = t - 18 * TY; ej = (u < 16) ? 0 : TY + 1; ei = 1 + (u & 15); }
                const int c = (ej + 2) * NP + (ei + 2);
                T Uf[3][2][NV], dU[NV];
#pragma unroll
                for (int d = 0; d < 3; ++d) {
                    T Wm[NV], Wp[NV];
#pragma unroll
                    for (int v = 0; v < NV; ++v) {
                        const T* q = Pz[R] + v * G::PLN + c;
                        if (d == 0) face_values<T, RECON, EXT, fixed_theta(EXT, RECON)>(q, 1, Wm[v], Wp[v], ph);
                        else if (d == 1) face_values<T, RECON, EXT, fixed_theta(EXT, RECON)>(q, NP, Wm[v], Wp[v], ph);
                        else {
                            const int o = v * G::PLN + c;
                            if (RECON == PPM)
                                face_values5<T, RECON, EXT>(Pz[0][o], Pz[R - 1][o], Pz[R][o], Pz[R + 1][o], Pz[2 * R][o], Wm[v], Wp[v], ph);
                            else
                                face_values5<T, RECON, EXT>(T(0), Pz[R - 1][o], Pz[R][o], Pz[R + 1][o], T(0), Wm[v], Wp[v], ph);
                        }
                    }
                    prim2cons<T, NV>(Wm, Uf[d][0], ph);
                    prim2cons<T, NV>(Wp, Uf[d][1], ph);
                    // F_d(W+) - F_d(W-), each difference formed as one product and one fused multiply-add
                    const T vm = Wm[1 + d], vp = Wp[1 + d];
                    T dF[NV];
#pragma unroll
                    for (int v = 0; v < NV; ++v) {
                        const T am = (v == 4) ? Uf[d][0][4] + Wm[4] : Uf[d][0][v];
                        const T ap = (v == 4) ? Uf[d][1][4] + Wp[4] : Uf[d][1][v];
                        dF[v] = ap * vp - am * vm;
                    }
                    dF[1 + d] += Wp[4] - Wm[4];
#pragma unroll
                    for (int v = 0; v < NV; ++v) dU[v] = (d == 0) ? dF[v] : dU[v] + dF[v];
                }
                // Hancock half step on all six face states, back to primitives, positivity check
                T We[3][2][NV];
                bool ok = true;
#pragma unroll
                for (int d = 0; d < 3; ++d)
#pragma unroll
                    for (int s = 0; s < 2; ++s) {
                        T Ue[NV];
#pragma unroll
                        for (int v = 0; v < NV; ++v) Ue[v] = Uf[d][s][v] - ph.hlam * dU[v];
                        cons2prim<T, NV>(Ue, We[d][s], ph);
                        if (EXT && ph.floors) floor_prim(We[d][s], ph);
                        ok = ok && (We[d][s][0] > T(0)) && (We[d][s][4] > T(0));
                    }
                if (!ok) {   // revert the cell's six states to the un-evolved face values
                    cnt.reverted++;
#pragma unroll
                    for (int d = 0; d < 3; ++d)
#pragma unroll
                        for (int s = 0; s < 2; ++s) cons2prim<T, NV>(Uf[d][s], We[d][s], ph);
                }
                const int e = ej * G::EW + ei;
                // rotated storage: array of axis d holds (rho, v_d, v_{d+1}, v_{d+2}, P [, q])
#pragma unroll
                for (int k = 0; k < NV; ++k) {
                    es[(0 * NV + k) * G::EPL + e] = We[0][0][nat_index(0, k)];
                    es[(1 * NV + k) * G::EPL + e] = We[0][1][nat_index(0, k)];
                    es[(2 * NV + k) * G::EPL + e] = We[1][0][nat_index(1, k)];
                    es[(3 * NV + k) * G::EPL + e] = We[1][1][nat_index(1, k)];
                    es[(4 * NV + k) * G::EPL + e] = We[2][0][nat_index(2, k)];
                    zcur[k * G::EPL + e] = We[2][1][nat_index(2, k)];
                }
            }
        }
        __syncthreads();
        // ------------------------------------------------------------------ S2: Riemann + convert next plane
        {
            const int f_lo = (kk >= 0 && kk < PS) ? 0 : G::NFX + G::NFY;
            const int f_hi = (kk >= 0 && kk <= PS) ? G::NF : 0;
            const int zpar = ((kk + 1) & 1) * NV * G::EPL;      // z+ states of plane kk-1
#pragma unroll
            for (int r = 0; r < NROUND; ++r) {
                const int f = tid + r * NT;
                if (f >= f_lo && f < f_hi)
                    cnt.roe_fb += riemann_face_rot<T, SOLVER, NV, TY>(es, fl, gflux, fdesc[r], f, zpar, kk, j0, ph);
            }
        }
        {
            const int n = kk + 2 + 2 * R;
            if (n < NPL) {
                mbar_wait(&bars[n & 1], (n >> 1) & 1);
                convert_plane<T, NV, EXT, TY, NT>(raw + (n & 1) * NV * G::PLN, prim + ((PF + n) % PR) * NV * G::PLN, ph, ctid);
            }
        }
        __syncthreads();
        // ------------------------------------------------------------------ S3: update plane kk-1, prepare plane kk
        if (tid == 0) {
            const int n = kk + 4 + 2 * R;
            if (n < NPL) issue_plane<T, NV, TY>(gin, j0, PF + n, raw + (n & 1) * NV * G::PLN, &bars[n & 1]);
        }
        if (owner && kk >= 1) {
            const int k = kk - 1;
            const T* gcell = gin + (size_t)(k + NGH) * (NP * NP) + (j0 + cj + NGH) * NP + (ci + NGH);
            T U[NV];
#pragma unroll
            for (int v = 0; v < NV; ++v) {
                const T dfz = fl[rot_index(2, v) * G::NF + G::NFX + G::NFY + tid] - fzm[v];
                U[v] = __ldg(gcell + (size_t)v * NPC) - ph.lam * (sxy[v] + dfz);
            }
            close_cell<T, SOLVER, NV, EXT>(U, gcell, cnt, ph);
#pragma unroll
            for (int v = 0; v < NV; ++v) gout[((size_t)v * PS + k) * (PS * PS) + (j0 + cj) * PS + ci] = U[v];
            if (a.speed) {
                const T s = signal_speed<T, NV, MHM, EXT>(U, ph);
                if (s > smax) smax = s;
            }
        }
        if (owner && kk >= 0 && kk < PS) {
#pragma unroll
            for (int v = 0; v < NV; ++v) {
                const T* px = fl + rot_index(0, v) * G::NF + cj * 17 + ci;
                const T* py = fl + rot_index(1, v) * G::NF + G::NFX + cj * 16 + ci;
                const T dfx = px[1] - px[0];
                const T dfy = py[16] - py[0];
                sxy[v] = dfx + dfy;
                fzm[v] = fl[rot_index(2, v) * G::NF + G::NFX + G::NFY + tid];
            }
        }
    }

    block_epilogue<T, NT, G::NTILE, EXT>(a, g, smax, cnt, sm, tid);
}

}  // namespace gamer
