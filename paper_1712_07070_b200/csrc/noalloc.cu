// noalloc.cu -- gamer_fluid_advance_table_noalloc: one step from the UNPADDED state + same-level neighbour table through a
// padded batch that lives in a file-scope static device array, for callers that cannot call cudaMalloc (code under CUDA graph
// capture, tight serving loops, harnesses that forbid allocation).  See include/gamer_hydro.h for the contract.
//
// What the existing path does with caller-provided scratch (gamer_refresh_ghosts_table into a padded batch the caller
// allocated, then gamer_fluid_advance_ex on it) is done here with the scratch below; the two kernels are the same, so
// the results carry the same bits.  Unlike gamer_fluid_advance_resident (no scratch at all, ghost zones gathered inside
// the solver) this form keeps the padded slab in memory, which is what remedy (ii) of PAPER.md L105 re-reads: it is the
// allocation-free way to run remedy_first_order from an unpadded state.
#include <cmath>
#include <mutex>

#include "../../include/gamer_hydro.h"
#include <cuda_runtime.h>

namespace {

// The padded batch [n_groups][NVAR][22][22][22].  64 MiB: 315 groups at NVAR = 5 in fp32, 157 in fp64 (1.3e6 / 6.4e5
// cells -- the batch size at which the paper's solvers saturate).  Every GPU that loads the library holds
// these bytes until the process exits.
static __device__ __align__(256) unsigned char g_padded_scratch[GAMER_NOALLOC_SCRATCH_BYTES];

// In host code `g_padded_scratch` is a host-side stand-in, not a device address: the address a kernel may use comes
// from cudaGetSymbolAddress, asked once per device with that device current.
constexpr int MAX_DEVICES = 64;
void* g_scratch_ptr[MAX_DEVICES] = {};
std::mutex g_scratch_mu;

int scratch_address(void** out) {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= MAX_DEVICES) return GAMER_ECUDA;
    std::lock_guard<std::mutex> lock(g_scratch_mu);
    if (!g_scratch_ptr[dev]) {
        void* p = nullptr;
        if (cudaGetSymbolAddress(&p, g_padded_scratch) != cudaSuccess || !p) return GAMER_ECUDA;
        g_scratch_ptr[dev] = p;
    }
    *out = g_scratch_ptr[dev];
    return GAMER_OK;
}

}  // namespace

extern "C" int64_t gamer_noalloc_max_groups(int nvar, int precision) {
    if (nvar < 5 || nvar > 5 + GAMER_MAX_SCALARS || (precision != GAMER_FP32 && precision != GAMER_FP64)) return 0;
    return (int64_t)(GAMER_NOALLOC_SCRATCH_BYTES / ((size_t)nvar * 22 * 22 * 22 * (size_t)precision));
}

extern "C" int gamer_fluid_advance_table_noalloc(const void* u, const int32_t* nbr, void* out, void* flux_out, int64_t n_groups,
                                                 double dt, double dh, double gamma, int scheme, int recon, int riemann,
                                                 int precision, const gamer_opts* opts) {
    if (n_groups < 0 || (n_groups > 0 && (!u || !nbr || !out)) || u == out) return GAMER_EINVAL;
    if (precision != GAMER_FP32 && precision != GAMER_FP64) return GAMER_EINVAL;
    const int nsc = opts ? opts->n_scalar : 0;
    if (nsc < 0 || nsc > GAMER_MAX_SCALARS) return GAMER_EINVAL;
    const int nvar = 5 + nsc;
    if (n_groups > gamer_noalloc_max_groups(nvar, precision)) return GAMER_ETOOLARGE;      // beyond the static scratch
    if (n_groups == 0) return GAMER_OK;
    void* padded = nullptr;
    int rc = scratch_address(&padded);
    if (rc) return rc;
    void* stream = opts ? opts->stream : nullptr;
    // The array keeps the last call's contents.  Slabs whose table entry is -1 are not written by the refresh (they are the
    // caller's to fill in the allocating path); here nobody else can fill them, so they start from zero rather than from
    // whatever an earlier call left: the result never depends on the call before.
    const size_t bytes = (size_t)n_groups * nvar * 22 * 22 * 22 * (size_t)precision;
    if (cudaMemsetAsync(padded, 0, bytes, static_cast<cudaStream_t>(stream)) != cudaSuccess) return GAMER_ECUDA;
    rc = gamer_refresh_ghosts_table(u, padded, nbr, n_groups, nvar, precision, stream);
    if (rc) return rc;
    return gamer_fluid_advance_ex(padded, out, flux_out, n_groups, dt, dh, gamma, scheme, recon, riemann, precision, opts);
}
