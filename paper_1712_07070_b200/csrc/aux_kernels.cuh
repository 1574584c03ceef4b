// aux_kernels.cuh -- CFL reduction (Eqs. 1-2) and the device-side
// same-level ghost refresh (the paper's CPU "preparation" step for sibling copies, L248).
#pragma once
#include "hydro_close.cuh"

namespace gamer {

__device__ __forceinline__ void atomic_max_nonneg(double* addr, double v) {
    // non-negative IEEE doubles order like their bit patterns; max is order-independent, so the
    // reduction stays bitwise reproducible
    atomicMax(reinterpret_cast<unsigned long long*>(addr), (unsigned long long)__double_as_longlong(v));
}

template <typename T> struct CflArgs {
    const T* u;
    T* speed;        // nullable
    double* acc;     // device double holding the running max (bits), zeroed before the launch
    double gamma, min_dens, min_pres, min_temp;
    long long n_groups;
};

// one CTA per patch group, 256 threads, 16 cells per thread, 16-byte loads
template <typename T, int NV, int SCHEME>
__global__ void __launch_bounds__(256) cfl_kernel(const CflArgs<T> a) {
    constexpr int NC = PS * PS * PS;
    constexpr int VEC = 16 / sizeof(T);
    Phys<T> ph;
    ph.gamma = T(a.gamma); ph.gm1 = T(a.gamma - 1.0); ph.inv_gm1 = T(1.0 / (a.gamma - 1.0));
    ph.min_dens = T(a.min_dens); ph.min_pres = T(a.min_pres); ph.min_temp = T(a.min_temp);
    ph.floors = (a.min_dens > 0.0 || a.min_pres > 0.0 || a.min_temp > 0.0) ? 1 : 0;
    const long long g = blockIdx.x;
    const T* base = a.u + (size_t)g * NV * NC;
    T smax = T(0);
    for (int c = threadIdx.x * VEC; c < NC; c += 256 * VEC) {
        T U[NV][VEC];
#pragma unroll
        for (int v = 0; v < NV; ++v) {
            if constexpr (sizeof(T) == 4) {
                const float4 q = __ldg(reinterpret_cast<const float4*>(base + (size_t)v * NC + c));
                U[v][0] = q.x; U[v][1] = q.y; U[v][2] = q.z; U[v][3] = q.w;
            } else {
                const double2 q = __ldg(reinterpret_cast<const double2*>(base + (size_t)v * NC + c));
                U[v][0] = q.x; U[v][1] = q.y;
            }
        }
#pragma unroll
        for (int e = 0; e < VEC; ++e) {
            T Uc[NV];
#pragma unroll
            for (int v = 0; v < NV; ++v) Uc[v] = U[v][e];
            const T s = signal_speed<T, NV, SCHEME, true>(Uc, ph);
            if (s > smax) smax = s;
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const T other = __shfl_xor_sync(0xffffffffu, smax, o);
        smax = other > smax ? other : smax;
    }
    __shared__ T red[8];
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = smax;
    __syncthreads();
    if (threadIdx.x == 0) {
        T m = red[0];
#pragma unroll
        for (int w = 1; w < 8; ++w) m = red[w] > m ? red[w] : m;
        if (a.speed) a.speed[g] = m;
        atomic_max_nonneg(a.acc, (double)m);
    }
}

// max over the per-group maxima -> running max (bits) in *acc
template <typename T>
__global__ void __launch_bounds__(1024) group_max_kernel(const T* speed, long long n, double* acc) {
    T m = T(0);
    for (long long i = blockIdx.x * 1024ll + threadIdx.x; i < n; i += 1024ll * gridDim.x) {
        const T s = speed[i];
        if (s > m) m = s;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const T other = __shfl_xor_sync(0xffffffffu, m, o);
        m = other > m ? other : m;
    }
    __shared__ T red[32];
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = m;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < 32; ++w) m = red[w] > m ? red[w] : m;
        atomic_max_nonneg(acc, (double)m);
    }
}

// *acc holds the max speed: replace it by dt = cfl*dh/max
__global__ void finish_dt_kernel(double* acc, double cfl_dh) { *acc = cfl_dh / *acc; }

// padded `in` batch from the unpadded `u` batch of a periodic box of gz x gy x gx groups.
// One CTA per (group, variable): 256 threads own two (row, column) positions of the 22 x 22 plane each and
// walk the 22 planes; the wrapped source offset splits into a per-thread (x,y) part computed once and a
// per-plane (z) part that is uniform over the CTA.  Writes are fully contiguous (a padded variable block is
// 10,648 consecutive elements), reads are 16-element rows of the neighbours' unpadded blocks.
template <typename T>
__global__ void __launch_bounds__(256) refresh_periodic_kernel(const T* __restrict__ u, T* __restrict__ in, int gz,
                                                               int gy, int gx, int nvar) {
    const long long gv = blockIdx.x;
    const long long g = gv / nvar;
    const int v = (int)(gv - g * nvar);
    const int bx = (int)(g % gx), by = (int)((g / gx) % gy), bz = (int)(g / ((long long)gx * gy));
    const size_t gstride = (size_t)nvar * (PS * PS * PS);
    size_t offxy[2];
    bool live[2];
#pragma unroll
    for (int r = 0; r < 2; ++r) {
        const int t = threadIdx.x + r * 256;
        live[r] = t < NP * NP;
        const int pj = t / NP, pi = t - pj * NP;
        int sx = bx, lx = pi - NGH, sy = by, ly = pj - NGH;
        if (lx < 0) { lx += PS; sx = sx == 0 ? gx - 1 : sx - 1; } else if (lx >= PS) { lx -= PS; sx = sx == gx - 1 ? 0 : sx + 1; }
        if (ly < 0) { ly += PS; sy = sy == 0 ? gy - 1 : sy - 1; } else if (ly >= PS) { ly -= PS; sy = sy == gy - 1 ? 0 : sy + 1; }
        offxy[r] = ((size_t)sy * gx + sx) * gstride + (size_t)v * (PS * PS * PS) + ly * PS + lx;
    }
    T* dst = in + ((size_t)g * nvar + v) * NPC;
    for (int pk = 0; pk < NP; ++pk) {
        int sz = bz, lz = pk - NGH;
        if (lz < 0) { lz += PS; sz = sz == 0 ? gz - 1 : sz - 1; } else if (lz >= PS) { lz -= PS; sz = sz == gz - 1 ? 0 : sz + 1; }
        const size_t offz = (size_t)sz * gy * gx * gstride + (size_t)lz * (PS * PS);
#pragma unroll
        for (int r = 0; r < 2; ++r)
            if (live[r]) dst[pk * (NP * NP) + threadIdx.x + r * 256] = __ldg(u + offz + offxy[r]);
    }
}

// neighbour table of a periodic box of gz x gy x gx groups: nbr[g][(dz+1)*9 + (dy+1)*3 + (dx+1)]
__global__ void neighbors_periodic_kernel(int* __restrict__ nbr, int gz, int gy, int gx) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long ng = (long long)gz * gy * gx;
    if (i >= ng * 27) return;
    const long long g = i / 27;
    const int k = (int)(i - g * 27);
    const int dx = k % 3 - 1, dy = (k / 3) % 3 - 1, dz = k / 9 - 1;
    const int bx = (int)(g % gx), by = (int)((g / gx) % gy), bz = (int)(g / ((long long)gx * gy));
    const int sx = (bx + dx + gx) % gx, sy = (by + dy + gy) % gy, sz = (bz + dz + gz) % gz;
    nbr[i] = (int)(((long long)sz * gy + sy) * gx + sx);
}

}  // namespace gamer
