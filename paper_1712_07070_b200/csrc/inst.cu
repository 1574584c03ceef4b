// inst.cu -- one translation unit per (scheme, recon, riemann): compiled 12 times with
// -DG_SCHEME=.. -DG_RECON=.. -DG_SOLVER=..; each instantiates fp32/fp64 x {fast, extended, extended+scalar}.
#include "launch.cuh"

#ifndef G_SCHEME
#error "compile with -DG_SCHEME=1|2|3 -DG_RECON=1|2 -DG_SOLVER=1|2|3|4 (scheme 3 = VL: recon 1 only)"
#endif

#define G_CAT2(a, b, c, d) a##b##_##c##_##d
#define G_CAT(a, b, c, d) G_CAT2(a, b, c, d)
#define G_NAME G_CAT(gamer_launch_, G_SCHEME, G_RECON, G_SOLVER)

namespace gamer {

template <typename T, int NV, bool EXT>
static cudaError_t go(const void* args, cudaStream_t st, int* launches) {
    const AdvArgs<T>& a = *static_cast<const AdvArgs<T>*>(args);
#if G_SCHEME == 1
    return launch_mhm<T, G_RECON, G_SOLVER, NV, EXT>(a, st, launches);
#elif G_SCHEME == 3
    return launch_mhm<T, G_RECON, G_SOLVER, NV, EXT, true>(a, st, launches);
#elif defined(GAMER_HAVE_CTU)
    return launch_ctu<T, G_RECON, G_SOLVER, NV, EXT>(a, st, launches);
#else
    (void)a; (void)st; (void)launches;
    return cudaErrorNotSupported;
#endif
}

template <typename T>
static cudaError_t by_scalars(int nsc, int ext, const void* args, cudaStream_t st, int* launches) {
    switch (nsc) {
    case 0: return ext ? go<T, 5, true>(args, st, launches) : go<T, 5, false>(args, st, launches);
    case 1: return go<T, 6, true>(args, st, launches);
    case 2: return go<T, 7, true>(args, st, launches);
    case 3: return go<T, 8, true>(args, st, launches);
    case 4: return go<T, 9, true>(args, st, launches);
    default: return cudaErrorNotSupported;
    }
}

// prec = 4|8, nsc = 0..4 passive scalars, ext = 0|1 (nsc > 0 implies ext)
cudaError_t G_NAME(int prec, int nsc, int ext, const void* args, cudaStream_t st, int* launches) {
    return prec == 4 ? by_scalars<float>(nsc, ext, args, st, launches) : by_scalars<double>(nsc, ext, args, st, launches);
}

}  // namespace gamer
