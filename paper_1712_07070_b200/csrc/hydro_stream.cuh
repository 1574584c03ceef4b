// hydro_stream.cuh -- shared machinery of the z-streaming patch-group kernels.
//
// One CTA advances one (16 x TY x 16) column tile of a patch group (TY = 16 is the whole group),
// marching along z one plane at a time.  Padded conserved planes are staged in shared memory with
// 1-D TMA bulk copies (cp.async.bulk + mbarrier, two stages in flight), converted to primitives
// into a ring of 2R+1 planes (R = reconstruction radius), and every intermediate of the scheme
// (face states, fluxes) lives only in shared memory / registers for the planes in flight, so HBM
// sees the algorithmic bytes only: one read of `in`, one write of `out` / `flux_out`.
// (The paper's own kernels kept these intermediates in global memory.)
#pragma once
#include "hydro_riemann.cuh"

namespace gamer {

constexpr int PS = 16;   // cells per patch-group edge
constexpr int NGH = 3;   // ghost zones (L300)
constexpr int NP = 22;   // padded edge
constexpr int NPC = NP * NP * NP;

template <typename T> struct AdvArgs {
    const T* in;
    T* out;
    T* flux;          // nullable
    T* speed;         // nullable
    int* n_unphys;    // nullable
    int* diag;        // nullable, int[4]
    const double* dt_dev;
    const int* nbr;   // nullable: [n_groups][27] same-level neighbour table => `in` is the UNPADDED state (fused refresh)
    double dt, dh, gamma, theta, xi, min_dens, min_pres, min_temp;
    int limiter, dual, remedy2, char_limit, renorm;
    long long n_groups;
    Phys<T> ph;       // the run-time constants in the kernel's precision, filled on the host (fill_phys)
};

// host side: every constant of the step in the kernel's precision, so that device code reads them straight
// from the kernel-parameter constant bank (no per-use double -> T conversion, no registers)
template <typename T>
inline void fill_phys(AdvArgs<T>& a) {
    Phys<T>& ph = a.ph;
    const double lam = a.dt / a.dh;
    ph.gamma = T(a.gamma);
    ph.gm1 = T(a.gamma - 1.0);
    ph.inv_gm1 = T(1.0 / (a.gamma - 1.0));
    ph.lam = T(lam);
    ph.hlam = T(0.5 * lam);
    ph.theta = T(a.theta);
    ph.limiter = a.limiter;
    ph.xi = T(a.xi);
    ph.min_dens = T(a.min_dens);
    ph.min_pres = T(a.min_pres);
    ph.min_temp = T(a.min_temp);
    ph.floors = (a.min_dens > 0.0 || a.min_pres > 0.0 || a.min_temp > 0.0) ? 1 : 0;
    ph.dual = a.dual;
    ph.remedy2 = a.remedy2;
    ph.char_limit = a.char_limit;
    ph.renorm = a.renorm;
}

// device side: the host-filled constants; only dt/dh comes from memory when dt lives on the device
template <typename T>
__device__ __forceinline__ Phys<T> make_phys(const AdvArgs<T>& a) {
    Phys<T> ph = a.ph;
    if (a.dt_dev) {
        const double lam = *a.dt_dev / a.dh;
        ph.lam = T(lam);
        ph.hlam = T(0.5 * lam);
    }
    return ph;
}

// ---------------------------------------------------------------------------------------------
// TMA 1-D bulk copy + mbarrier (sm_90+ PTX; SASS: UBLKCP / SYNCS)
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    uint32_t ok = 0;
    const uint32_t addr = smem_u32(bar);
    while (!ok) {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(ok)
            : "r"(addr), "r"(parity)
            : "memory");
    }
}
__device__ __forceinline__ void tma_load_1d(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
            smem_u32(dst)),
        "l"(src), "r"(bytes), "r"(smem_u32(bar))
        : "memory");
}
__device__ __forceinline__ void fence_proxy_async() {
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}

// ---------------------------------------------------------------------------------------------
// tile geometry
// ---------------------------------------------------------------------------------------------
template <int TY> struct Geo {
    static constexpr int NT = 16 * TY;            // threads per CTA = cells per plane of the tile
    static constexpr int NTILE = PS / TY;         // tiles per group
    static constexpr int NR = TY + 2 * NGH;       // rows of a staged plane
    static constexpr int PLN = NR * NP;           // elements of a staged plane (per variable)
    static constexpr int EW = 18, EH = TY + 2;    // face-state plane: cells -1..16 x -1..TY
    static constexpr int EPL = EW * EH;
    static constexpr int NPLUS = 18 * TY + 32;    // cells whose face states the final pass needs
    static constexpr int NFX = 17 * TY, NFY = 16 * (TY + 1), NFZ = 16 * TY;
    static constexpr int NF = NFX + NFY + NFZ;
};

// stage the padded conserved plane p (0..21) of the tile into raw stage `st`
template <typename T, int NV, int TY>
__device__ __forceinline__ void issue_plane(const T* gin, int j0, int p, T* raw_stage, uint64_t* bar) {
    using G = Geo<TY>;
    constexpr uint32_t bytes = G::PLN * sizeof(T);
    fence_proxy_async();
    mbar_expect_tx(bar, bytes * NV);
#pragma unroll
    for (int v = 0; v < NV; ++v)
        tma_load_1d(raw_stage + v * G::PLN, gin + (size_t)v * NPC + (size_t)p * (NP * NP) + j0 * NP, bytes, bar);
}

// raw conserved plane -> primitive plane (O1), floors in extended mode
template <typename T, int NV, bool EXT, int TY, int NT = Geo<TY>::NT>
__device__ __forceinline__ void convert_plane(const T* raw, T* prim, const Phys<T>& ph, int tid) {
    using G = Geo<TY>;
    for (int t = tid; t < G::PLN; t += NT) {
        T U[NV], W[NV];
#pragma unroll
        for (int v = 0; v < NV; ++v) U[v] = raw[v * G::PLN + t];
        cons2prim<T, NV>(U, W, ph);
        if (EXT && ph.floors) floor_prim(W, ph);
#pragma unroll
        for (int v = 0; v < NV; ++v) prim[v * G::PLN + t] = W[v];
    }
}

// ---------------------------------------------------------------------------------------------
// Fused ghost refresh: the padded plane is gathered straight from the
// unpadded state of the group and of its same-level neighbours with cp.async (LDGSTS), so no padded copy of the
// batch ever exists in HBM.  Staged rows are 24 wide with the 16 interior cells at columns 4..19 (16-byte aligned
// for the wide copies), ghosts at 1..3 and 20..22 (columns 0 and 23 receive a fourth, unused neighbour cell so that
// the ghost cells travel as aligned 16-byte chunks too).  nb = the 27 neighbour group indices of this group.
// ---------------------------------------------------------------------------------------------
constexpr int FW = 24;   // row stride of a staged plane in fused mode

__device__ __forceinline__ void cp_async_16(void* dst, const void* src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
// wait until at most N of this thread's committed copy groups are still in flight
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// One copy of the gather of a padded plane: destination element inside the landing stage, source element inside a
// group's plane z (v*16^3 + y*16 + x), which in-plane neighbour (dy*3 + dx) holds it, and whether it is a 16-byte
// copy.  The list is the same for every plane: each thread decodes its few entries once (stage_plane_fused_regs).
template <typename T, int NV, int TY> struct FusedCopies {
    static constexpr int CE = 16 / (int)sizeof(T);          // elements per 16-byte copy
    static constexpr int GC = 4 / CE;                       // copies per ghost side: the 3 ghost cells travel as the
                                                            // aligned 4-element chunk that contains them
    static constexpr int OPS = PS / CE + 2 * GC;            // copies per row and variable, all 16 bytes wide
    static constexpr int N = Geo<TY>::NR * NV * OPS;
};

// entry `it` of the copy list: .x = destination element in the landing stage, .y = source element | in-plane neighbour << 20
template <typename T, int NV, int TY>
__device__ __forceinline__ int2 fused_copy_desc(int it, int j0) {
    using G = Geo<TY>;
    using F = FusedCopies<T, NV, TY>;
    constexpr int PS3 = PS * PS * PS;
    const int op = it % F::OPS, rv = it / F::OPS;
    const int r = rv % G::NR, v = rv / G::NR;
    const int py = j0 + r;
    const int dy = py < NGH ? 0 : (py < NGH + PS ? 1 : 2);
    const int yy = (py + PS - NGH) & (PS - 1);
    int dx, xx, col;
    if (op < PS / F::CE) { dx = 1; xx = op * F::CE; col = 4 + xx; }                      // interior cells
    else if (op < PS / F::CE + F::GC) { dx = 0; xx = PS - 4 + (op - PS / F::CE) * F::CE; col = xx - (PS - 4); }   // x' 12..15 -> cols 0..3
    else { dx = 2; xx = (op - PS / F::CE - F::GC) * F::CE; col = 4 + PS + xx; }           // x' 0..3 -> cols 20..23
    return make_int2((v * G::NR + r) * FW + col, (v * PS3 + yy * PS + xx) | ((dy * 3 + dx) << 20));
}

// Every thread issues its own entries of the list for padded plane p (0..21) and commits them as one cp.async group.  The
// entries (NCP = ceil(N / nthr) per thread, .x < 0 = none) are the same for every plane, so each thread decodes its own once,
// keeps them in registers, and the per-plane work is one table look-up (neighbour group), one 64-bit address and the copy per entry.
template <typename T, int NV, int NCP>
__device__ __forceinline__ void stage_plane_fused_regs(const T* u, const int* nb, const int2 (&cd)[NCP], int p, T* raw_stage) {
    constexpr int PS3 = PS * PS * PS;
    const int dz = p < NGH ? 0 : (p < NGH + PS ? 1 : 2);
    const int zoff = ((p + PS - NGH) & (PS - 1)) * (PS * PS);
    const int* nbz = nb + dz * 9;
#pragma unroll
    for (int i = 0; i < NCP; ++i) {
        if (cd[i].x >= 0) {
            const T* src = u + (size_t)nbz[cd[i].y >> 20] * NV * PS3 + ((cd[i].y & 0xfffff) + zoff);
            cp_async_16(raw_stage + cd[i].x, src);
        }
    }
    cp_async_commit();
}

// raw conserved plane in the fused layout -> primitive plane in the standard [NV][NR*22] layout
template <typename T, int NV, bool EXT, int TY, int NT>
__device__ __forceinline__ void convert_plane_fused(const T* raw, T* prim, const Phys<T>& ph, int tid) {
    using G = Geo<TY>;
    for (int t = tid; t < G::PLN; t += NT) {
        const int r = t / NP, cx = t - r * NP;
        T U[NV], W[NV];
#pragma unroll
        for (int v = 0; v < NV; ++v) U[v] = raw[(v * G::NR + r) * FW + cx + 1];
        cons2prim<T, NV>(U, W, ph);
        if (EXT && ph.floors) floor_prim(W, ph);
#pragma unroll
        for (int v = 0; v < NV; ++v) prim[v * G::PLN + t] = W[v];
    }
}

template <typename T, int RECON, bool EXT>
__device__ __forceinline__ void face_values5(T l2, T l1, T c, T r1, T r2, T& wm, T& wp, const Phys<T>& ph) {
    T q[5] = {l2, l1, c, r1, r2};
    face_values<T, RECON, EXT, fixed_theta(EXT, RECON)>(q + 2, 1, wm, wp, ph);
}

// ---------------------------------------------------------------------------------------------
// face states / fluxes in shared memory as one 16-byte vector + NV-4 scalars
// ---------------------------------------------------------------------------------------------
template <typename T> struct alignas(16) Vec4 {
    T a, b, c, d;
};

template <typename T> struct alignas(16) Vec2 {
    T a, b;
};

// five (six) values of one face <-> shared memory: one Vec4 + NV-4 scalars; n = entries of the array.
// fp64: a 32-byte Vec4 per lane is two 16-byte accesses at stride 32 -- every quarter-warp spans 256 bytes, a 2-way bank
// conflict on each -- so the four values are kept as two arrays of 16-byte pairs [Vec2 n | Vec2 n | (NV-4) x n] in the same space.
template <typename T, int NV>
__device__ __forceinline__ void put_state(T* blk, int n, int idx, const T* W) {
    if constexpr (sizeof(T) == 8) {
        Vec2<T> lo, hi;
        lo.a = W[0]; lo.b = W[1]; hi.a = W[2]; hi.b = W[3];
        reinterpret_cast<Vec2<T>*>(blk)[idx] = lo;
        reinterpret_cast<Vec2<T>*>(blk + 2 * n)[idx] = hi;
#pragma unroll
        for (int v = 4; v < NV; ++v) blk[v * n + idx] = W[v];
        return;
    }
    Vec4<T> q;
    q.a = W[0]; q.b = W[1]; q.c = W[2]; q.d = W[3];
    reinterpret_cast<Vec4<T>*>(blk)[idx] = q;
#pragma unroll
    for (int v = 4; v < NV; ++v) blk[v * n + idx] = W[v];
}
template <typename T, int NV>
__device__ __forceinline__ void get_state(const T* blk, int n, int idx, T* W) {
    if constexpr (sizeof(T) == 8) {
        const Vec2<T> lo = reinterpret_cast<const Vec2<T>*>(blk)[idx];
        const Vec2<T> hi = reinterpret_cast<const Vec2<T>*>(blk + 2 * n)[idx];
        W[0] = lo.a; W[1] = lo.b; W[2] = hi.a; W[3] = hi.b;
#pragma unroll
        for (int v = 4; v < NV; ++v) W[v] = blk[v * n + idx];
        return;
    }
    const Vec4<T> q = reinterpret_cast<const Vec4<T>*>(blk)[idx];
    W[0] = q.a; W[1] = q.b; W[2] = q.c; W[3] = q.d;
#pragma unroll
    for (int v = 4; v < NV; ++v) W[v] = blk[v * n + idx];
}


// ---------------------------------------------------------------------------------------------
// Rotated storage: a face-state array of axis d holds (rho, v_d, v_{d+1}, v_{d+2}, P [, q]) -- the producer rotates
// at compile time -- so the Riemann stage needs no per-face rotation arithmetic.
// rot_index(d, v) = position of natural variable v in the rotation of axis d; nat_index is its inverse.
// ---------------------------------------------------------------------------------------------
__host__ __device__ constexpr int rot_index(int d, int v) { return (v >= 1 && v <= 3) ? 1 + ((v - 1 - d + 3) % 3) : v; }
__host__ __device__ constexpr int nat_index(int d, int k) { return (k >= 1 && k <= 3) ? 1 + ((k - 1 + d) % 3) : k; }

}  // namespace gamer
