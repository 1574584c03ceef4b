// hydro_close.cuh -- closing step of one updated cell (PAPER.md L100 dual energy, L102-105 remedies,
// L504 floors) and the CFL signal speed (Eqs. 1-2).
#pragma once
#include "hydro_stream.cuh"

namespace gamer {

template <typename T, int NV>
__device__ __forceinline__ bool is_physical(const T* U) {
    bool ok = U[0] > T(0);
#pragma unroll
    for (int v = 0; v < NV; ++v) ok = ok && Ops<T>::finite(U[v]);
    const T ek = T(0.5) * (U[1] * U[1] + U[2] * U[2] + U[3] * U[3]) / U[0];
    return ok && (U[4] - ek) > T(0);
}

// E_the/E_kin < xi: rebuild E from the entropy; otherwise resynchronise the entropy from E (L100)
template <typename T, int NV>
__device__ __forceinline__ int dual_energy_fix(T* U, const Phys<T>& ph) {
    if (NV < 6 || !ph.dual || !(U[0] > T(0))) return 0;
    const T ek = T(0.5) * (U[1] * U[1] + U[2] * U[2] + U[3] * U[3]) / U[0];
    const T et = U[4] - ek;
    const T rg = Ops<T>::pow(U[0], ph.gm1);
    if (et < ph.xi * ek) {
        U[4] = ek + U[NV - 1] * rg * ph.inv_gm1;
        return 1;
    }
    U[NV - 1] = ph.gm1 * et / rg;
    return 0;
}

template <typename T, int NV>
__device__ __forceinline__ void floor_cons(T* U, const Phys<T>& ph) {
    if (ph.min_dens > T(0) && U[0] < ph.min_dens) U[0] = ph.min_dens;
    const T ek = T(0.5) * (U[1] * U[1] + U[2] * U[2] + U[3] * U[3]) / U[0];
    const T P = ph.gm1 * (U[4] - ek);
    T pf = ph.min_pres;
    const T pt = U[0] * ph.min_temp;
    if (pt > pf) pf = pt;
    if (pf > T(0) && P < pf) {
        U[4] = ek + pf * ph.inv_gm1;
        if (NV > 5 && ph.dual) U[NV - 1] = pf / Ops<T>::pow(U[0], ph.gm1);
    }
}

// L96: the passive scalars (all but the entropy of the dual-energy formalism, which is the last one) rescaled so that they
// sum to rho; a non-positive sum is left alone (DESIGN R27)
template <typename T, int NV>
__device__ __forceinline__ void renormalize_scalars(T* U, const Phys<T>& ph) {
    if (NV < 6 || !ph.renorm) return;
    const int last = NV - (ph.dual ? 1 : 0);
    T sum = T(0);
#pragma unroll
    for (int v = 5; v < NV; ++v)
        if (v < last) sum = sum + U[v];
    if (!(sum > T(0))) return;
    const T f = U[0] / sum;
#pragma unroll
    for (int v = 5; v < NV; ++v)
        if (v < last) U[v] = U[v] * f;
}

// running maximum of the CFL signal speeds.  A NaN speed (a cell that came out with P < 0) never wins the comparison, as
// in the oracle's reduction: such cells are what n_unphysical_out counts and remedies (iv)/(v) act on; the time-step
// of the remaining cells stays usable for the retry.
template <typename T>
__device__ __forceinline__ T speed_max(T smax, T s) { return s > smax ? s : smax; }

template <typename T, int NV, int SCHEME, bool EXT>
__device__ __forceinline__ T signal_speed(const T* U, const Phys<T>& ph) {
    T W[NV];
    cons2prim<T, NV>(U, W, ph);
    if (EXT && ph.floors) floor_prim(W, ph);
    const T cs = Ops<T>::sqrt(ph.gamma * W[4] * Ops<T>::rcp(W[0]));
    const T ax = Ops<T>::abs(W[1]), ay = Ops<T>::abs(W[2]), az = Ops<T>::abs(W[3]);
    if (SCHEME == MHM) return ax + ay + az + T(3) * cs;
    return Ops<T>::max(Ops<T>::max(ax, ay), az) + cs;
}

// remedy (ii), L105: first order in space and time, unsplit, same Riemann solver, straight from the
// padded input in global memory (rare path).  gin points at variable 0 of the padded cell.
template <typename T, int SOLVER, int NV, bool EXT>
__device__ __noinline__ void first_order_cell(const T* gin, T* Unew, int* nfb, const Phys<T>& ph) {
    T Uc[NV], Wc[NV], acc[NV];
#pragma unroll
    for (int v = 0; v < NV; ++v) { Uc[v] = gin[(size_t)v * NPC]; acc[v] = T(0); }
    cons2prim<T, NV>(Uc, Wc, ph);
    const int step[3] = {1, NP, NP * NP};
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const int cn = 1 + d, c1 = 1 + (d + 1) % 3, c2 = 1 + (d + 2) % 3;
        T Wr[NV] ;
        Wr[0] = Wc[0]; Wr[1] = Wc[cn]; Wr[2] = Wc[c1]; Wr[3] = Wc[c2]; Wr[4] = Wc[4];
#pragma unroll
        for (int v = 5; v < NV; ++v) Wr[v] = Wc[v];
        T Fd[NV];
#pragma unroll
        for (int v = 0; v < NV; ++v) Fd[v] = T(0);
#pragma unroll
        for (int s = 0; s < 2; ++s) {
            T Un[NV], Wn[NV], Wq[NV], F[NV];
            const int off = s ? step[d] : -step[d];
#pragma unroll
            for (int v = 0; v < NV; ++v) Un[v] = gin[(size_t)v * NPC + off];
            cons2prim<T, NV>(Un, Wn, ph);
            Wq[0] = Wn[0]; Wq[1] = Wn[cn]; Wq[2] = Wn[c1]; Wq[3] = Wn[c2]; Wq[4] = Wn[4];
#pragma unroll
            for (int v = 5; v < NV; ++v) Wq[v] = Wn[v];
            const bool fb = s ? riemann_flux<T, SOLVER, NV>(Wr, Wq, F, ph) : riemann_flux<T, SOLVER, NV>(Wq, Wr, F, ph);
            *nfb += fb ? 1 : 0;
            const T sg = s ? T(1) : T(-1);
            Fd[0] += sg * F[0];
            Fd[cn] += sg * F[1];
            Fd[c1] += sg * F[2];
            Fd[c2] += sg * F[3];
            Fd[4] += sg * F[4];
#pragma unroll
            for (int v = 5; v < NV; ++v) Fd[v] += sg * F[v];
        }
#pragma unroll
        for (int v = 0; v < NV; ++v) acc[v] += Fd[v];
    }
#pragma unroll
    for (int v = 0; v < NV; ++v) Unew[v] = Uc[v] - ph.lam * acc[v];
}

struct Counters {
    int roe_fb, reverted, first_order, dual_fix, unphys;
};

// finish one interior cell: U holds the high-order update on entry, the final state on exit
template <typename T, int SOLVER, int NV, bool EXT>
__device__ __forceinline__ void close_cell(T* U, const T* gin_cell, Counters& cnt, const Phys<T>& ph) {
    if (!EXT) return;
    cnt.dual_fix += dual_energy_fix<T, NV>(U, ph);
    if (ph.remedy2 && !is_physical<T, NV>(U)) {
        cnt.first_order++;
        first_order_cell<T, SOLVER, NV, EXT>(gin_cell, U, &cnt.roe_fb, ph);
        cnt.dual_fix += dual_energy_fix<T, NV>(U, ph);
    }
    if (ph.floors) floor_cons<T, NV>(U, ph);
    renormalize_scalars<T, NV>(U, ph);
    if (!is_physical<T, NV>(U)) cnt.unphys++;
}

// block epilogue shared by the kernels: per-group CFL maximum (warp shuffles -> smem -> one value; atomicMax on
// the bit pattern only when a group is split in tiles) and the integer diagnostics
template <typename T, int NT, int NTILE, bool EXT>
__device__ __forceinline__ void block_epilogue(const AdvArgs<T>& a, long long g, T smax, const Counters& cnt, T* red, int tid) {
    __syncthreads();
    if (a.speed) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const T other = __shfl_xor_sync(0xffffffffu, smax, o);
            smax = other > smax ? other : smax;
        }
        if ((tid & 31) == 0) red[tid >> 5] = smax;
        __syncthreads();
        if (tid == 0) {
            T mx = red[0];
            for (int w = 1; w < NT / 32; ++w) mx = red[w] > mx ? red[w] : mx;
            if (NTILE == 1) a.speed[g] = mx;
            else if (sizeof(T) == 4) atomicMax(reinterpret_cast<unsigned int*>(a.speed + g), __float_as_uint((float)mx));
            else atomicMax(reinterpret_cast<unsigned long long*>(a.speed + g), (unsigned long long)__double_as_longlong((double)mx));
        }
    }
    if (EXT) {
        int c[5] = {cnt.roe_fb, cnt.reverted, cnt.first_order, cnt.dual_fix, cnt.unphys};
#pragma unroll
        for (int q = 0; q < 5; ++q) {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) c[q] += __shfl_xor_sync(0xffffffffu, c[q], o);
        }
        if ((tid & 31) == 0) {
            if (a.diag) {
                if (c[0]) atomicAdd(a.diag + 0, c[0]);
                if (c[1]) atomicAdd(a.diag + 1, c[1]);
                if (c[2]) atomicAdd(a.diag + 2, c[2]);
                if (c[3]) atomicAdd(a.diag + 3, c[3]);
            }
            if (a.n_unphys && c[4]) atomicAdd(a.n_unphys, c[4]);
        }
    }
}

}  // namespace gamer
