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
    int nvar;        // variables per cell in u (5 + passive scalars); only the first five enter the signal speed
};

// one CTA per patch group, 256 threads, 16 cells per thread, 16-byte loads
template <typename T, int SCHEME>
__global__ void __launch_bounds__(256) cfl_kernel(const CflArgs<T> a) {
    constexpr int NC = PS * PS * PS;
    constexpr int VEC = 16 / sizeof(T);
    Phys<T> ph;
    ph.gamma = T(a.gamma); ph.gm1 = T(a.gamma - 1.0); ph.inv_gm1 = T(1.0 / (a.gamma - 1.0));
    ph.min_dens = T(a.min_dens); ph.min_pres = T(a.min_pres); ph.min_temp = T(a.min_temp);
    ph.floors = (a.min_dens > 0.0 || a.min_pres > 0.0 || a.min_temp > 0.0) ? 1 : 0;
    const long long g = blockIdx.x;
    constexpr int NV = 5;
    const T* base = a.u + (size_t)g * a.nvar * NC;
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
            smax = speed_max(smax, s);
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

// Same-level ghost refresh of a uniform level with the boundary conditions of PAPER.md L98 per face:
// 0 periodic, 1 outflow (zero gradient: nearest cell inside), 2 reflecting (mirror cell, normal momentum negated).
// One CTA per (group, variable) as refresh_periodic_kernel; bc = {x_lo, x_hi, y_lo, y_hi, z_lo, z_hi}.
struct BcSet { int v[6]; };

// global cell index c (may lie outside [0, n)) -> source cell; *flip is set when the cell is a mirror image
__device__ __forceinline__ int bc_source(int c, int n, int lo, int hi, bool* flip) {
    *flip = false;
    if (c >= 0 && c < n) return c;
    const int kind = c < 0 ? lo : hi;
    if (kind == 1) return c < 0 ? 0 : n - 1;
    if (kind == 2) { *flip = true; return c < 0 ? -1 - c : 2 * n - 1 - c; }
    return c < 0 ? c + n : c - n;
}

template <typename T>
__global__ void __launch_bounds__(256) refresh_bc_kernel(const T* __restrict__ u, T* __restrict__ in, int gz, int gy,
                                                         int gx, int nvar, BcSet bc) {
    const long long gv = blockIdx.x;
    const long long g = gv / nvar;
    const int v = (int)(gv - g * nvar);
    const int bx = (int)(g % gx), by = (int)((g / gx) % gy), bz = (int)(g / ((long long)gx * gy));
    const size_t gstride = (size_t)nvar * (PS * PS * PS);
    size_t offxy[2];
    bool live[2], neg[2];
#pragma unroll
    for (int r = 0; r < 2; ++r) {
        const int t = threadIdx.x + r * 256;
        live[r] = t < NP * NP;
        const int pj = t / NP, pi = t - pj * NP;
        bool fx, fy;
        const int cx = bc_source(bx * PS + pi - NGH, gx * PS, bc.v[0], bc.v[1], &fx);
        const int cy = bc_source(by * PS + pj - NGH, gy * PS, bc.v[2], bc.v[3], &fy);
        neg[r] = (v == 1 && fx) != (v == 2 && fy);      // at most one of the two can be true for a given v
        offxy[r] = ((size_t)(cy / PS) * gx + cx / PS) * gstride + (size_t)v * (PS * PS * PS) + (cy % PS) * PS + (cx % PS);
    }
    T* dst = in + ((size_t)g * nvar + v) * NPC;
    for (int pk = 0; pk < NP; ++pk) {
        bool fz;
        const int cz = bc_source(bz * PS + pk - NGH, gz * PS, bc.v[4], bc.v[5], &fz);
        const size_t offz = (size_t)(cz / PS) * gy * gx * gstride + (size_t)(cz % PS) * (PS * PS);
        const bool nz = (v == 3 && fz);
#pragma unroll
        for (int r = 0; r < 2; ++r)
            if (live[r]) {
                const T val = __ldg(u + offz + offxy[r]);
                dst[pk * (NP * NP) + threadIdx.x + r * 256] = (neg[r] != nz) ? -val : val;
            }
    }
}

// Same-level ghost refresh driven by a neighbour table (any topology): one CTA per (group, variable); padded cell
// (pk, pj, pi) comes from the group nbr[g][(dz*3 + dy)*3 + dx] named for its slab, or is left untouched if that entry
// is -1 (coarse-fine boundary, filled by the caller's interpolation).
template <typename T>
__global__ void __launch_bounds__(256) refresh_table_kernel(const T* __restrict__ u, T* __restrict__ in,
                                                            const int* __restrict__ nbr, int nvar) {
    __shared__ int nb[27];
    const long long gv = blockIdx.x;
    const long long g = gv / nvar;
    const int v = (int)(gv - g * nvar);
    if (threadIdx.x < 27) nb[threadIdx.x] = nbr[g * 27 + threadIdx.x];
    __syncthreads();
    int offxy[2], sxy[2];
    bool live[2];
#pragma unroll
    for (int r = 0; r < 2; ++r) {
        const int t = threadIdx.x + r * 256;
        live[r] = t < NP * NP;
        const int pj = t / NP, pi = t - pj * NP;
        const int dx = pi < NGH ? 0 : (pi < NGH + PS ? 1 : 2), dy = pj < NGH ? 0 : (pj < NGH + PS ? 1 : 2);
        sxy[r] = dy * 3 + dx;
        offxy[r] = ((pj + PS - NGH) & (PS - 1)) * PS + ((pi + PS - NGH) & (PS - 1));
    }
    T* dst = in + ((size_t)g * nvar + v) * NPC;
    for (int pk = 0; pk < NP; ++pk) {
        const int dz = pk < NGH ? 0 : (pk < NGH + PS ? 1 : 2);
        const int offz = ((pk + PS - NGH) & (PS - 1)) * (PS * PS);
#pragma unroll
        for (int r = 0; r < 2; ++r)
            if (live[r]) {
                const int s = nb[dz * 9 + sxy[r]];
                if (s >= 0) dst[pk * (NP * NP) + threadIdx.x + r * 256] = __ldg(u + ((size_t)s * nvar + v) * (PS * PS * PS) + offz + offxy[r]);
            }
    }
}

// Ghost zones at coarse-fine boundaries "interpolat[ed] from coarse patches", linear in time between the
// coarse level's two stored states (L482); R24: conservative piecewise-linear interpolation of the conserved
// variables, child = U_c + ((+-s_z) + (+-s_y) + (+-s_x)) / 4 with central or minmod slopes.  One CTA per (fine group,
// variable); only the slabs whose entry of the fine level's neighbour table is negative are written.  Fine padded index p
// along an axis -> fine cell i = p - 3 -> coarse cell 8 o + floor(i / 2) of the parent group (padded index + 3), child i & 1.
__device__ __forceinline__ double blend_rn(double w0, double a, double w1, double b) { return __dadd_rn(__dmul_rn(w0, a), __dmul_rn(w1, b)); }
__device__ __forceinline__ float blend_rn(float w0, float a, float w1, float b) { return __fadd_rn(__fmul_rn(w0, a), __fmul_rn(w1, b)); }

// Work is organised by coarse cell in y and z and by FINE cell in x: u and the three limited slopes are formed once per
// (coarse z, coarse y, fine x) item and serve its four (ck, cj) children, whose signs are compile-time constants of the
// unrolled loops, and consecutive lanes write consecutive fine cells.  (The first version walked the 22^3 fine cells and
// rebuilt the slopes for every one of them: 99 instructions per ghost value, issue-bound at 27 % of the HBM roof; a version
// with all eight children per thread wrote every other cell of a row per store: 6.5 sectors per request.)
constexpr int INTERP_NT = 288;

template <typename T, bool BLEND, bool MONO>
__global__ void __launch_bounds__(INTERP_NT) interpolate_ghosts_kernel(const T* __restrict__ c0, const T* __restrict__ c1, T w0, T w1,
                                                                       T* __restrict__ fine, const int* __restrict__ parent,
                                                                       const int* __restrict__ nbr, int nvar) {
    __shared__ int nb[27];
    const long long gv = blockIdx.x;
    const long long g = gv / nvar;
    const int v = (int)(gv - g * nvar);
    if (threadIdx.x < 27) nb[threadIdx.x] = nbr[g * 27 + threadIdx.x];
    __syncthreads();
    bool any = false;
#pragma unroll
    for (int s = 0; s < 27; ++s) any = any || (s != 13 && nb[s] < 0);
    if (!any) return;                                  // no coarse-fine slab in this group (uniform over the CTA)
    const int par = parent[g];
    const int oz = (par >> 2) & 1, oy = (par >> 1) & 1, ox = par & 1;
    const size_t cbase = ((size_t)(par >> 3) * nvar + v) * NPC;
    const T* a0 = c0 + cbase;
    const T* a1 = BLEND ? c1 + cbase : nullptr;
    T* dst = fine + ((size_t)g * nvar + v) * NPC;
    // the 14^3 coarse cells under this octant's ghost zones (+1 for the slopes), blended in time once: padded coarse
    // indices 8 o .. 8 o + 13 along each axis; a thread carries one (j, i) of the block through its 14 planes
    constexpr int CB = 14;
    __shared__ T cs[CB * CB * CB];
    for (int t = threadIdx.x; t < CB * CB; t += INTERP_NT) {
        const int j = t / CB, i = t - j * CB;
        const int q0 = ((8 * oz) * NP + 8 * oy + j) * NP + 8 * ox + i;
#pragma unroll
        for (int k = 0; k < CB; ++k) {
            const T x = __ldg(a0 + q0 + k * (NP * NP));
            cs[k * (CB * CB) + t] = BLEND ? blend_rn(w0, x, w1, __ldg(a1 + q0 + k * (NP * NP))) : x;
        }
    }
    __syncthreads();
    auto slope = [&](T lo, T mid, T hi) -> T {
        if (!MONO) return T(0.5) * (hi - lo);
        const T a = mid - lo, b = hi - mid;
        return a * b > T(0) ? (fabs(a) < fabs(b) ? a : b) : T(0);
    };
    // Staged coarse index l = 1..12 along an axis holds the fine padded cells p = 2l - 3 (child 0) and 2l - 2 (child 1):
    // l = 1, 2 are the low ghost zones (p = 0 | 1, 2), l = 3..10 the interior, l = 11, 12 the high ones (p = 19, 20 | 21);
    // p = -1 and p = 22 do not exist.  Both children of a coarse cell lie in the same slab of the neighbour table.
    // Work items = (coarse z, coarse y, fine x) triples of the ghost shell only, in three segments: the four z-ghost
    // coarse planes in full (4 x 12 x 22), the four y-ghost coarse rows of the eight inner planes (8 x 4 x 22), the six
    // x-ghost fine columns of their inner rows (8 x 8 x 6).  2144 items of four children each (6552 ghost cells, plus the
    // children at p = -1 / 22 that do not exist) instead of 12 x 12 x 22 with the interior masked out.
    constexpr int NA = 4 * 12 * NP, NB = 8 * 4 * NP, NC = 8 * 8 * 6;
    for (int it = threadIdx.x; it < NA + NB + NC; it += INTERP_NT) {
        int lk, lj, pi;
        if (it < NA) {
            const int a = it / (12 * NP), r = it - a * (12 * NP);
            lk = a < 2 ? a + 1 : a + 9;
            lj = r / NP + 1;
            pi = r - (lj - 1) * NP;
        } else if (it < NA + NB) {
            const int r = it - NA, a = r / (4 * NP), r2 = r - a * (4 * NP), c = r2 / NP;
            lk = a + 3;
            lj = c < 2 ? c + 1 : c + 9;
            pi = r2 - c * NP;
        } else {
            const int r = it - NA - NB, a = r / 48, r2 = r - a * 48, c = r2 / 6, x = r2 - c * 6;
            lk = a + 3;
            lj = c + 3;
            pi = x < 3 ? x : x + 16;
        }
        const int li = ((pi + 1) >> 1) + 1;
        const bool ui = (pi + 1) & 1;
        const int dz = lk < 3 ? 0 : (lk < 11 ? 1 : 2), dy = lj < 3 ? 0 : (lj < 11 ? 1 : 2), dx = li < 3 ? 0 : (li < 11 ? 1 : 2);
        if (nb[dz * 9 + dy * 3 + dx] >= 0) continue;
        const int q = (lk * CB + lj) * CB + li;
        const T u = cs[q];
        const T sz = slope(cs[q - CB * CB], u, cs[q + CB * CB]);
        const T sy = slope(cs[q - CB], u, cs[q + CB]);
        const T sx = slope(cs[q - 1], u, cs[q + 1]);
        const T sxs = ui ? sx : -sx;
        const int pk0 = 2 * lk - 3, pj0 = 2 * lj - 3;
#pragma unroll
        for (int ck = 0; ck < 2; ++ck) {
            const int pk = pk0 + ck;
            if (pk < 0 || pk >= NP) continue;
#pragma unroll
            for (int cj = 0; cj < 2; ++cj) {
                const int pj = pj0 + cj;
                if (pj < 0 || pj >= NP) continue;
                dst[(pk * NP + pj) * NP + pi] = u + T(0.25) * (((ck ? sz : -sz) + (cj ? sy : -sy)) + sxs);
            }
        }
    }
}

// Refined-level Poisson solver (R25): one CTA relaxes one patch's
// (8 + 2*5)^3 = 18^3 potential, held entirely in shared memory as the paper does (49.2 KB in fp64 with its padded rows), by red-black SOR with
// the outermost cells fixed; thread (k, j) owns row (k, j) of the 16^3 relaxed cells: 8 cells per colour, source term in
// registers.  Then the potential goes back and, optionally, -grad(phi) of the 8^3 active zones by central differences.
constexpr int PN = 18, PR = 16, PA0 = 5, PAN = 8;
// Row and plane stride of the potential in shared memory.  fp32: rows of 18, planes of 18 * 18 + 1 (= 1 mod 4), see the bank
// note below.  fp64: a lane's 8-byte access covers a pair of banks and a warp is served as two half-warps of 16 lanes = 2 plane
// indices k x 8 row indices j (stride 2, parity alternating with k).  With rows of 18 doubles two j-rows are 72 words apart:
// 72 m mod 32 takes only four values, rows m and m + 4 share their banks -- a 2-way conflict on every access (measured: 50 %
// excess wavefronts with the shared-memory pipe 95 % busy).  Rows of 19 doubles: 76 m mod 32 = 12 m = 0, 12, 24, 4, 16, 28, 8, 20,
// eight distinct bank pairs {4q, 4q+1}; the plane stride must then be EVEN (342): the next k is 684 +- 38 words on (its rows have
// the other parity) = 18 or 6 mod 32, the pairs {4q+2, 4q+3} -- one wavefront per half-warp.  (Checked with a 32-lane
// LDS.64 microbenchmark: 343 gives the 2-way conflict back.)
template <typename T> struct SorGeo {
    static constexpr int RS = sizeof(T) == 8 ? 19 : 18;                    // row stride
    static constexpr int PL = PN * RS + (sizeof(T) == 8 ? 0 : 1);          // plane stride: 325 (fp32), 342 (fp64)
    static constexpr size_t BYTES = (size_t)PN * PL * sizeof(T);
};

// One half-sweep over the cells i = 2 - IP, 4 - IP, ... of the thread's row: x-neighbours from the row's registers, the four
// others from shared memory, the new value to both.  Same order of additions as the oracle.
template <typename T, int IP>
__device__ __forceinline__ void sor_half_sweep(T (&me)[PN], const T (&src)[PR], T* row, T w6) {
#pragma unroll
    for (int m = 0; m < PR / 2; ++m) {
        constexpr int dummy = 0; (void)dummy;
        const int i = 2 - IP + 2 * m;
        constexpr int RS = SorGeo<T>::RS, PL = SorGeo<T>::PL;
        const T r = me[i - 1] + me[i + 1] + row[i - RS] + row[i + RS] + row[i - PL] + row[i + PL] - T(6) * me[i] - src[i - 1];
        me[i] += w6 * r;
        row[i] = me[i];
    }
}

// Thread layout: warps 0-3 own the rows with (j + k) even, warps 4-7 those with (j + k) odd, so the x-parity of a colour's
// cells is uniform over a warp and the row can live in registers with static indices.  Lane -> (k, j): r = (warp & 3) * 32 + lane,
// k = 1 + r / 8, j = 1 + 2 (r % 8) + s with s fixing the parity.  Banks (fp32): 4 k + 4 (r % 8) + 18 s + i with the padded plane
// stride (= 1 mod 4) puts the 32 lanes of a warp on 32 different banks.
// (poisson_sor_kernel below, after the gravity helpers it calls.)

// Fluid gravity update of one cell (DESIGN R28): U points at variable 0 of the cell in the patch-group
// layout (variable stride 16^3); momentum kick dt * rho * g, energy by the kinetic-energy difference.
template <typename T>
__device__ __forceinline__ void gravity_kick(T* U, T ax, T ay, T az, T dt) {
    constexpr int VS = PS * PS * PS;
    const T rho = U[0], mx = U[VS], my = U[2 * VS], mz = U[3 * VS];
    const T k = dt * rho;
    const T nx = mx + k * ax, ny = my + k * ay, nz = mz + k * az;
    const T ke_new = (nx * nx + ny * ny) + nz * nz, ke_old = (mx * mx + my * my) + mz * mz;
    U[4 * VS] = U[4 * VS] + T(0.5) * (ke_new - ke_old) / rho;
    U[VS] = nx; U[2 * VS] = ny; U[3 * VS] = nz;
}

// the cell (ai, aj, ak) of patch n's 8^3 active zones inside the patch-group batch: patch n = 8 g + oz*4 + oy*2 + ox
__device__ __forceinline__ size_t patch_cell_in_group(size_t n, int nvar, int ak, int aj, int ai) {
    const size_t g = n >> 3;
    const int o = (int)(n & 7);
    return g * nvar * (PS * PS * PS) + (size_t)(((o >> 2) * 8 + ak) * PS + (((o >> 1) & 1) * 8 + aj)) * PS + ((o & 1) * 8 + ai);
}

template <typename T>
__global__ void __launch_bounds__(256) gravity_update_kernel(T* __restrict__ flu, const T* __restrict__ acc, int nvar, T dt) {
    const size_t n = blockIdx.x;
    const T* ga = acc + n * (3 * 512);
    for (int t = threadIdx.x; t < 512; t += 256)
        gravity_kick(flu + patch_cell_in_group(n, nvar, t >> 6, (t >> 3) & 7, t & 7), ga[t], ga[t + 512], ga[t + 1024], dt);
}

template <typename T>
__global__ void __launch_bounds__(256) poisson_sor_kernel(T* __restrict__ phi, const T* __restrict__ rho, T* __restrict__ acc,
                                                          T* __restrict__ resid, T src_scale, T w6, T inv_2dh, int n_iter,
                                                          T* __restrict__ flu = nullptr, int nvar = 0, T dt_g = T(0)) {
    constexpr int RS = SorGeo<T>::RS, PL = SorGeo<T>::PL;
    extern __shared__ __align__(16) unsigned char sor_smem[];      // SorGeo<T>::BYTES (fp64: 49.2 KB, above the static limit)
    T* p = reinterpret_cast<T*>(sor_smem);
    const size_t n = blockIdx.x;
    T* gp = phi + n * (PN * PN * PN);
    for (int t = threadIdx.x; t < PN * PN * PN; t += 256) {
        const int kk = t / (PN * PN), rr = t - kk * (PN * PN), jj = rr / PN;
        p[kk * PL + jj * RS + (rr - jj * PN)] = gp[t];
    }
    const int par = threadIdx.x >> 7, r = threadIdx.x & 127;
    const int k = 1 + (r >> 3), j = 1 + 2 * (r & 7) + ((par + k + 1) & 1);
    T src[PR], me[PN];
    const T* gr = rho + n * (PR * PR * PR) + (size_t)((k - 1) * PR + (j - 1)) * PR;
#pragma unroll
    for (int i = 0; i < PR; ++i) src[i] = src_scale * gr[i];
    __syncthreads();
    T* row = p + k * PL + j * RS;
#pragma unroll
    for (int i = 0; i < PN; ++i) me[i] = row[i];
    for (int it = 0; it < n_iter; ++it) {
        // colour 0 = cells with (i + j + k) even: i even in the even rows, odd in the odd rows; then colour 1
        if (par) sor_half_sweep<T, 1>(me, src, row, w6); else sor_half_sweep<T, 0>(me, src, row, w6);
        __syncthreads();
        if (par) sor_half_sweep<T, 0>(me, src, row, w6); else sor_half_sweep<T, 1>(me, src, row, w6);
        __syncthreads();
    }
    if (resid) {
        // defect of the discretised equation after the last iteration, max over the patch (order-independent: reproducible)
        __shared__ T wmax[8];
        T m = T(0);
#pragma unroll
        for (int i = 1; i <= PR; ++i)
            m = fmax(m, fabs(me[i - 1] + me[i + 1] + row[i - RS] + row[i + RS] + row[i - PL] + row[i + PL] - T(6) * me[i] - src[i - 1]));
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
        if ((threadIdx.x & 31) == 0) wmax[threadIdx.x >> 5] = m;
        __syncthreads();
        if (threadIdx.x == 0) {
#pragma unroll
            for (int w = 1; w < 8; ++w) m = fmax(m, wmax[w]);
            resid[n] = m;
        }
    }
    for (int t = threadIdx.x; t < PN * PN * PN; t += 256) {
        const int kk = t / (PN * PN), rr = t - kk * (PN * PN), jj = rr / PN;
        gp[t] = p[kk * PL + jj * RS + (rr - jj * PN)];
    }
    if (acc || flu) {      // acceleration of the active zones; the fluid's gravity update straight from it (L238)
        T* ga = acc ? acc + n * (3 * PAN * PAN * PAN) : nullptr;
        for (int t = threadIdx.x; t < PAN * PAN * PAN; t += 256) {
            const int ak = t / (PAN * PAN), aj = (t / PAN) % PAN, ai = t % PAN;
            const T* c = p + (ak + PA0) * PL + (aj + PA0) * RS + ai + PA0;
            const T ax = -(c[1] - c[-1]) * inv_2dh, ay = -(c[RS] - c[-RS]) * inv_2dh, az = -(c[PL] - c[-PL]) * inv_2dh;
            if (ga) {
                ga[t] = ax;
                ga[t + PAN * PAN * PAN] = ay;
                ga[t + 2 * PAN * PAN * PAN] = az;
            }
            if (flu) gravity_kick(flu + patch_cell_in_group(n, nvar, ak, aj, ai), ax, ay, az, dt_g);
        }
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

// ---------------------------------------------------------------------------------------------
// fix-up between a refined patch group and the coarse level
// ---------------------------------------------------------------------------------------------
// restriction: one CTA per (fine group, variable), one thread per coarse cell of the 8^3 octant; the eight children
// are added in the order (dz, dy, dx) = (0,0,0), (0,0,1), ... and scaled by 1/8
template <typename T>
__global__ void __launch_bounds__(512) restrict_kernel(const T* __restrict__ fine, T* __restrict__ coarse,
                                                       const int* __restrict__ parent, int nvar) {
    const long long gv = blockIdx.x;
    const long long g = gv / nvar;
    const int v = (int)(gv - g * nvar);
    const int par = parent[g];
    const int oz = (par >> 2) & 1, oy = (par >> 1) & 1, ox = par & 1;
    const int t = threadIdx.x, i = t & 7, j = (t >> 3) & 7, k = t >> 6;
    const T* f = fine + ((size_t)g * nvar + v) * (PS * PS * PS) + ((2 * k) * PS + 2 * j) * PS + 2 * i;
    T s = T(0);
#pragma unroll
    for (int dz = 0; dz < 2; ++dz)
#pragma unroll
        for (int dy = 0; dy < 2; ++dy) {
            // two neighbouring fine cells in one vector load
            const T a = f[(dz * PS + dy) * PS], b = f[(dz * PS + dy) * PS + 1];
            s = s + a;
            s = s + b;
        }
    coarse[((size_t)(par >> 3) * nvar + v) * (PS * PS * PS) + ((oz * 8 + k) * PS + (oy * 8 + j)) * PS + (ox * 8 + i)] = T(0.125) * s;
}

// acc = (init ? 0 : acc) + w * flux, elementwise (time average of the fine flux_out over the sub-steps)
template <typename T>
__global__ void flux_accumulate_kernel(T* __restrict__ acc, const T* __restrict__ flux, T w, long long n, int init) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        acc[i] = init ? w * flux[i] : acc[i] + w * flux[i];
}

// flux correction: one CTA per table entry (an 8 x 8 patch of coarse faces), thread = coarse face; only the entries
// of pass = axis * 2 + side act, so no two CTAs of a launch touch the same cell and the result is order-independent
template <typename T>
__global__ void __launch_bounds__(64) flux_correct_kernel(T* __restrict__ coarse, const T* __restrict__ coarse_flux,
                                                          const T* __restrict__ fine_flux_avg, const int* __restrict__ tab,
                                                          int nvar, T lam, int pass) {
    const int* e = tab + 8 * (size_t)blockIdx.x;
    const int d = e[1], side = e[2];
    if (d * 2 + side != pass) return;
    const T sgn = side ? T(1) : T(-1);
    const int b0 = e[5] >> 8, a0 = e[5] & 255;
    const int b = threadIdx.x >> 3, a = threadIdx.x & 7;
    int z = e[7] >> 16, y = (e[7] >> 8) & 255, x = e[7] & 255;
    if (d == 0) { z += b; y += a; } else if (d == 1) { z += b; x += a; } else { y += b; x += a; }
    for (int v = 0; v < nvar; ++v) {
        const T* ff = fine_flux_avg + ((((size_t)e[0] * 3 + d) * 3 + (side ? 2 : 0)) * nvar + v) * (PS * PS) + (2 * b) * PS + 2 * a;
        const T* fc = coarse_flux + ((((size_t)e[3] * 3 + d) * 3 + e[4]) * nvar + v) * (PS * PS);
        T* c = coarse + ((size_t)e[6] * nvar + v) * (PS * PS * PS) + (z * PS + y) * PS + x;
        const T favg = T(0.25) * (((ff[0] + ff[1]) + ff[PS]) + ff[PS + 1]);
        const T corr = lam * (favg - fc[(b0 + b) * PS + (a0 + a)]);
        *c += sgn * corr;
    }
}

}  // namespace gamer
