// launch.cuh -- host-side launch helpers: tile height selection by shared-memory fit, attribute setup.
// MHM_TY_OVERRIDE, MHM_FORCE_NSTG2, CTU_TY_OVERRIDE are tuning hooks for experiments
// (GAMER_EXTRA_DEFS of build.py); the shipped library is built without them.
#pragma once
#include <cstdlib>
#include "mhm_kernel.cuh"
#ifdef GAMER_HAVE_CTU
#include "ctu_kernel.cuh"
#include "ctu_wl_kernel.cuh"
#endif

namespace gamer {

constexpr size_t SMEM_LIMIT = 232448;   // 227 KB opt-in maximum per CTA on sm_100

constexpr size_t SM_SMEM = 233472;      // 228 KB of shared memory per SM, 1 KB of it reserved per resident CTA
constexpr int ctas_by_smem(size_t bytes) { return (int)(SM_SMEM / (bytes + 1024)); }

// CTAs of tile height TY that share an SM, with the number of landing stages launch_mhm_f would pick for it
template <typename T, int RECON, int NV, int TY, bool VLS, bool FUSED>
constexpr int mhm_ctas() {
    constexpr int c2 = ctas_by_smem(MhmGeo<T, RECON, NV, TY, 2, FUSED, VLS>::BYTES), c1 = ctas_by_smem(MhmGeo<T, RECON, NV, TY, 1, FUSED, VLS>::BYTES);
    return (!FUSED && c1 >= 2 && c2 < 2) ? c1 : c2;
}

// Tile height: the largest that fits -- unless the full 16-row tile leaves the SM to a single CTA (10 warps) and 8-row tiles
// fit twice (12 warps, 10 % more halo cells): measured +1.1 % (MHM+PLM fp64), +4 % (VL+PLM fp32).
template <typename T, int RECON, int NV, bool VLS, bool FUSED>
constexpr int mhm_tile() {
    if (MhmGeo<T, RECON, NV, 16, 2, FUSED, VLS>::BYTES <= SMEM_LIMIT)
        return (mhm_ctas<T, RECON, NV, 16, VLS, FUSED>() >= 2 || mhm_ctas<T, RECON, NV, 8, VLS, FUSED>() < 2) ? 16 : 8;
    return MhmGeo<T, RECON, NV, 8, 2, FUSED, VLS>::BYTES <= SMEM_LIMIT ? 8 : 4;
}

template <typename T, int RECON, int SOLVER, int NV, bool EXT, bool FUSED, bool VLS>
cudaError_t launch_mhm_f(const AdvArgs<T>& a, cudaStream_t st, int* launches) {
#ifdef MHM_TY_OVERRIDE
    constexpr int TY = MHM_TY_OVERRIDE;
#else
    constexpr int TY = mhm_tile<T, RECON, NV, VLS, FUSED>();
#endif
    // two landing stages unless dropping to one lets a second CTA share the SM
    constexpr int C2 = ctas_by_smem(MhmGeo<T, RECON, NV, TY, 2, FUSED, VLS>::BYTES), C1 = ctas_by_smem(MhmGeo<T, RECON, NV, TY, 1, FUSED, VLS>::BYTES);
#ifdef MHM_FORCE_NSTG2
    constexpr int NSTG = 2;
#else
    constexpr int NSTG = (!FUSED && C1 >= 2 && C2 < 2) ? 1 : 2;      // the fused gather is pipelined over two stages
#endif
    using G = MhmGeo<T, RECON, NV, TY, NSTG, FUSED, VLS>;
    if constexpr (G::BYTES > SMEM_LIMIT) {      // not even the 4-row tile fits (many scalars in fp64): not built
        (void)a; (void)st; (void)launches;
        return cudaErrorNotSupported;
    } else {
    constexpr int MINB = ctas_by_smem(G::BYTES) >= 2 ? 2 : 1;
    auto kern = mhm_kernel<T, RECON, SOLVER, NV, EXT, TY, NSTG, MINB, FUSED, VLS>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)G::BYTES);
    if (e != cudaSuccess) return e;
    if (G::NTILE > 1 && a.speed) {
        e = cudaMemsetAsync(a.speed, 0, sizeof(T) * a.n_groups, st);
        if (e != cudaSuccess) return e;
    }
    const long long grid = a.n_groups * G::NTILE;
    kern<<<(unsigned)grid, G::NT, G::BYTES, st>>>(a);
    *launches += 1;
    return cudaGetLastError();
    }
}

// a.nbr set => `in` is the unpadded state and the ghost refresh is fused into the staging loads
template <typename T, int RECON, int SOLVER, int NV, bool EXT, bool VLS = false>
cudaError_t launch_mhm(const AdvArgs<T>& a, cudaStream_t st, int* launches) {
    return a.nbr ? launch_mhm_f<T, RECON, SOLVER, NV, EXT, true, VLS>(a, st, launches)
                 : launch_mhm_f<T, RECON, SOLVER, NV, EXT, false, VLS>(a, st, launches);
}

#ifdef GAMER_HAVE_CTU
// fp32: the thread-owned kernel (ctu_kernel.cuh); fp64: the work-list kernel (ctu_wl_kernel.cuh), see its header
template <typename T, int RECON, int NV, int TY, bool FUSED>
struct CtuPick {
    using S32 = CtuSmem<T, RECON, NV, TY, FUSED>;
    using S64 = CtuWlSmem<T, RECON, NV, TY, FUSED>;
    static constexpr bool WL = sizeof(T) == 8;
    static constexpr size_t BYTES = WL ? S64::BYTES : S32::BYTES;
    static constexpr int NT = WL ? (48 * TY < 128 ? 128 : 48 * TY) : S32::NT;
};

template <typename T, int RECON, int NV, bool FUSED>
constexpr int ctu_tile() {
    return CtuPick<T, RECON, NV, 16, FUSED>::BYTES <= SMEM_LIMIT ? 16 : (CtuPick<T, RECON, NV, 8, FUSED>::BYTES <= SMEM_LIMIT ? 8 : 4);
}

template <typename T, int RECON, int SOLVER, int NV, bool EXT, bool FUSED>
cudaError_t launch_ctu_f(const AdvArgs<T>& a, cudaStream_t st, int* launches) {
#ifdef CTU_TY_OVERRIDE
    constexpr int TY = CTU_TY_OVERRIDE;
#else
    constexpr int TY = ctu_tile<T, RECON, NV, FUSED>();
#endif
    using G = Geo<TY>;
    using S = CtuPick<T, RECON, NV, TY, FUSED>;
    if constexpr (S::BYTES > SMEM_LIMIT) {      // not even the 4-row tile fits (many scalars in fp64): not built
        (void)a; (void)st; (void)launches;
        return cudaErrorNotSupported;
    } else {
    cudaError_t (*set)(const void*, cudaFuncAttribute, int) = cudaFuncSetAttribute;
    const void* kern;
    if constexpr (S::WL) kern = (const void*)ctu_wl_kernel<T, RECON, SOLVER, NV, EXT, TY, S::NT, FUSED>;
    else kern = (const void*)ctu_kernel<T, RECON, SOLVER, NV, EXT, TY, FUSED>;
    cudaError_t e = set(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)S::BYTES);
    if (e != cudaSuccess) return e;
    if (G::NTILE > 1 && a.speed) {
        e = cudaMemsetAsync(a.speed, 0, sizeof(T) * a.n_groups, st);
        if (e != cudaSuccess) return e;
    }
    const long long grid = a.n_groups * G::NTILE;
    void* args[] = {const_cast<AdvArgs<T>*>(&a)};
    e = cudaLaunchKernel(kern, dim3((unsigned)grid), dim3(S::NT), args, S::BYTES, st);
    if (e != cudaSuccess) return e;
    *launches += 1;
    return cudaGetLastError();
    }
}

// a.nbr set => `in` is the unpadded state and the ghost refresh is fused into the staging loads
template <typename T, int RECON, int SOLVER, int NV, bool EXT>
cudaError_t launch_ctu(const AdvArgs<T>& a, cudaStream_t st, int* launches) {
    return a.nbr ? launch_ctu_f<T, RECON, SOLVER, NV, EXT, true>(a, st, launches)
                 : launch_ctu_f<T, RECON, SOLVER, NV, EXT, false>(a, st, launches);
}
#endif

}  // namespace gamer
