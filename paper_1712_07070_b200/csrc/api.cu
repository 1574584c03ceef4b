// api.cu -- the C ABI of include/gamer_hydro.h: argument validation, dispatch over
// (scheme, recon, riemann, precision), auxiliary kernels, and the host-buffer entry.
#include <atomic>
#include <cmath>
#include <cstring>
#include <algorithm>
#include <mutex>
#include <vector>

#include "../../include/gamer_hydro.h"
#include "aux_kernels.cuh"

namespace gamer {
#define G_DECL(s, r, v) cudaError_t gamer_launch_##s##_##r##_##v(int, int, int, const void*, cudaStream_t, int*);
G_DECL(1, 1, 1) G_DECL(1, 1, 2) G_DECL(1, 1, 3) G_DECL(1, 1, 4) G_DECL(1, 2, 1) G_DECL(1, 2, 2) G_DECL(1, 2, 3) G_DECL(1, 2, 4)
G_DECL(2, 1, 1) G_DECL(2, 1, 2) G_DECL(2, 1, 3) G_DECL(2, 1, 4) G_DECL(2, 2, 1) G_DECL(2, 2, 2) G_DECL(2, 2, 3) G_DECL(2, 2, 4)
G_DECL(3, 1, 1) G_DECL(3, 1, 2) G_DECL(3, 1, 3) G_DECL(3, 1, 4)
#undef G_DECL
typedef cudaError_t (*launch_fn)(int, int, int, const void*, cudaStream_t, int*);
static const launch_fn TABLE[3][2][4] = {
    {{gamer_launch_1_1_1, gamer_launch_1_1_2, gamer_launch_1_1_3, gamer_launch_1_1_4},
     {gamer_launch_1_2_1, gamer_launch_1_2_2, gamer_launch_1_2_3, gamer_launch_1_2_4}},
    {{gamer_launch_2_1_1, gamer_launch_2_1_2, gamer_launch_2_1_3, gamer_launch_2_1_4},
     {gamer_launch_2_2_1, gamer_launch_2_2_2, gamer_launch_2_2_3, gamer_launch_2_2_4}},
    {{gamer_launch_3_1_1, gamer_launch_3_1_2, gamer_launch_3_1_3, gamer_launch_3_1_4},
     {nullptr, nullptr, nullptr, nullptr}}};      // VL + PPM: needs a fourth ghost zone
static std::atomic<long long> g_launches{0};
}  // namespace gamer

using namespace gamer;

static bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

static int check_common(const void* in, const void* out, int64_t n_groups, double dh, double gamma, int scheme,
                        int recon, int riemann, int precision) {
    if (n_groups < 0 || (n_groups > 0 && (!in || !out))) return GAMER_EINVAL;
    if (!(dh > 0.0) || !std::isfinite(dh) || !(gamma > 1.0) || !std::isfinite(gamma)) return GAMER_EINVAL;
    if (scheme != GAMER_MHM && scheme != GAMER_CTU && scheme != GAMER_VL) return GAMER_EINVAL;
    if (recon != GAMER_PLM && recon != GAMER_PPM) return GAMER_EINVAL;
    if (riemann < GAMER_ROE || riemann > GAMER_EXACT) return GAMER_EINVAL;
    if (precision != GAMER_FP32 && precision != GAMER_FP64) return GAMER_EINVAL;
    if (!aligned16(in) || !aligned16(out)) return GAMER_EINVAL;
    if (scheme == GAMER_VL && recon != GAMER_PLM) return GAMER_EUNSUPPORTED;
    return GAMER_OK;
}

template <typename T>
static int advance_typed(const void* in, void* out, void* flux_out, int64_t n_groups, double dt, double dh,
                         double gamma, int scheme, int recon, int riemann, const gamer_opts* o,
                         const int32_t* nbr = nullptr) {
    AdvArgs<T> a;
    std::memset(&a, 0, sizeof(a));
    a.nbr = nbr;
    a.in = static_cast<const T*>(in);
    a.out = static_cast<T*>(out);
    a.flux = static_cast<T*>(flux_out);
    a.dt = dt; a.dh = dh; a.gamma = gamma;
    a.n_groups = n_groups;
    a.limiter = LIM_GMINMOD;
    a.theta = recon == GAMER_PPM ? 2.0 : 1.0;
    a.xi = 1e-2;
    cudaStream_t st = nullptr;
    int nsc = 0, ext = 0;
    if (o) {
        st = static_cast<cudaStream_t>(o->stream);
        if (o->limiter != 0) a.limiter = o->limiter;
        if (o->minmod_theta > 0.0) a.theta = o->minmod_theta;
        if (o->de_xi > 0.0) a.xi = o->de_xi;
        a.min_dens = o->min_dens; a.min_pres = o->min_pres; a.min_temp = o->min_temp;
        a.dual = o->dual_energy; a.remedy2 = o->remedy_first_order; a.char_limit = o->char_limiting ? 1 : 0;
        a.renorm = (o->renormalize && o->n_scalar - (o->dual_energy ? 1 : 0) > 0) ? 1 : 0;
        a.dt_dev = o->dt_dev;
        a.speed = static_cast<T*>(o->group_speed_out);
        a.n_unphys = o->n_unphysical_out;
        a.diag = o->diag_out;
        nsc = o->n_scalar;
        const bool custom_theta = a.theta != (recon == GAMER_PPM ? 2.0 : 1.0);   // fast kernels fix theta at compile time
        ext = (nsc || a.renorm || a.dual || a.remedy2 || a.limiter != LIM_GMINMOD || custom_theta || a.char_limit || a.min_dens > 0 || a.min_pres > 0 ||
               a.min_temp > 0 || a.n_unphys || a.diag) ? 1 : 0;
    }
    if (a.n_unphys && cudaMemsetAsync(a.n_unphys, 0, sizeof(int), st) != cudaSuccess) return GAMER_ECUDA;
    if (a.diag && cudaMemsetAsync(a.diag, 0, 4 * sizeof(int), st) != cudaSuccess) return GAMER_ECUDA;
    if (n_groups == 0) return GAMER_OK;
    fill_phys(a);
    int launches = 0;
    const cudaError_t e = TABLE[scheme - 1][recon - 1][riemann - 1](sizeof(T), nsc, ext, &a, st, &launches);
    g_launches += launches;
    if (e == cudaErrorNotSupported) return GAMER_EUNSUPPORTED;      // combination not built (e.g. a tile that cannot fit)
    return e == cudaSuccess ? GAMER_OK : GAMER_ECUDA;
}

extern "C" int gamer_fluid_advance_ex(const void* in, void* out, void* flux_out, int64_t n_groups, double dt,
                                      double dh, double gamma, int scheme, int recon, int riemann, int precision,
                                      const gamer_opts* opts) {
    int rc = check_common(in, out, n_groups, dh, gamma, scheme, recon, riemann, precision);
    if (rc) return rc;
    const bool dev_dt = opts && opts->dt_dev;
    if (!dev_dt && (!(dt > 0.0) || !std::isfinite(dt))) return GAMER_EINVAL;
    if (flux_out && !aligned16(flux_out)) return GAMER_EINVAL;
    if (opts) {
        if (opts->n_scalar < 0 || opts->n_scalar > GAMER_MAX_SCALARS) return GAMER_EINVAL;
        if (opts->dual_energy && opts->n_scalar < 1) return GAMER_EINVAL;      // the entropy is the last scalar
        if (opts->limiter < 0 || opts->limiter > GAMER_LIMITER_VANALBADA) return GAMER_EINVAL;
        if (opts->minmod_theta > 0.0 && !(opts->minmod_theta >= 1.0 && opts->minmod_theta <= 2.0)) return GAMER_EINVAL;   // TVD range
        if (opts->min_dens < 0 || opts->min_pres < 0 || opts->min_temp < 0) return GAMER_EINVAL;
    }
    if (n_groups > 0x3fffffff) return GAMER_EUNSUPPORTED;
    return precision == GAMER_FP32
               ? advance_typed<float>(in, out, flux_out, n_groups, dt, dh, gamma, scheme, recon, riemann, opts)
               : advance_typed<double>(in, out, flux_out, n_groups, dt, dh, gamma, scheme, recon, riemann, opts);
}

extern "C" int gamer_fluid_advance(const void* in, void* out, void* flux_out, int64_t n_groups, double dt, double dh,
                                   double gamma, int scheme, int recon, int riemann, int precision) {
    return gamer_fluid_advance_ex(in, out, flux_out, n_groups, dt, dh, gamma, scheme, recon, riemann, precision,
                                  nullptr);
}

extern "C" int gamer_fluid_advance_retry(const void* in, void* out, void* flux_out, int64_t n_groups, double dt,
                                         double dh, double gamma, int scheme, int recon, int riemann, int precision,
                                         const gamer_opts* opts, double dt_ratio, double dt_min, double* dt_used_host,
                                         int32_t* n_retries_host) {
    if (!opts || !opts->n_unphysical_out || opts->dt_dev) return GAMER_EINVAL;
    if (!(dt > 0.0) || !std::isfinite(dt) || !(dt_min >= 0.0) || !(dt_ratio < 1.0)) return GAMER_EINVAL;
    if (!(dt_ratio > 0.0)) dt_ratio = 0.8;   // L107 "0.8 by default"
    cudaStream_t st = static_cast<cudaStream_t>(opts->stream);
    int32_t retries = 0;
    for (;;) {
        const int rc = gamer_fluid_advance_ex(in, out, flux_out, n_groups, dt, dh, gamma, scheme, recon, riemann,
                                              precision, opts);
        if (rc) return rc;
        int32_t bad = 0;
        if (n_groups > 0 &&
            (cudaMemcpyAsync(&bad, opts->n_unphysical_out, sizeof(bad), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
             cudaStreamSynchronize(st) != cudaSuccess))
            return GAMER_ECUDA;
        if (dt_used_host) *dt_used_host = dt;
        if (n_retries_host) *n_retries_host = retries;
        if (bad == 0) return GAMER_OK;
        dt *= dt_ratio;                      // remedy (iv): the whole batch again with the reduced step
        ++retries;
        if (dt < dt_min || retries > 200) return GAMER_EUNPHYSICAL;   // remedy (v): the caller's abort
    }
}

extern "C" int gamer_fluid_advance_resident(const void* u, const int32_t* nbr, void* out, void* flux_out, int64_t n_groups,
                                            double dt, double dh, double gamma, int scheme, int recon, int riemann,
                                            int precision, const gamer_opts* opts) {
    int rc = check_common(u, out, n_groups, dh, gamma, scheme, recon, riemann, precision);
    if (rc) return rc;
    if (n_groups > 0 && !nbr) return GAMER_EINVAL;
    const bool dev_dt = opts && opts->dt_dev;
    if (!dev_dt && (!(dt > 0.0) || !std::isfinite(dt))) return GAMER_EINVAL;
    if (flux_out && !aligned16(flux_out)) return GAMER_EINVAL;
    if (opts) {
        if (opts->n_scalar < 0 || opts->n_scalar > GAMER_MAX_SCALARS) return GAMER_EINVAL;
        if (opts->dual_energy && opts->n_scalar < 1) return GAMER_EINVAL;      // the entropy is the last scalar
        if (opts->limiter < 0 || opts->limiter > GAMER_LIMITER_VANALBADA) return GAMER_EINVAL;
        if (opts->minmod_theta > 0.0 && !(opts->minmod_theta >= 1.0 && opts->minmod_theta <= 2.0)) return GAMER_EINVAL;   // TVD range
        if (opts->min_dens < 0 || opts->min_pres < 0 || opts->min_temp < 0) return GAMER_EINVAL;
        if (opts->remedy_first_order) return GAMER_EUNSUPPORTED;   // remedy (ii) re-reads the padded slab
    }
    if (n_groups > 0x3fffffff / 27) return GAMER_EUNSUPPORTED;
    if (u == out) return GAMER_EINVAL;
    return precision == GAMER_FP32
               ? advance_typed<float>(u, out, flux_out, n_groups, dt, dh, gamma, scheme, recon, riemann, opts, nbr)
               : advance_typed<double>(u, out, flux_out, n_groups, dt, dh, gamma, scheme, recon, riemann, opts, nbr);
}

extern "C" int gamer_neighbors_periodic(int32_t* nbr, int gz, int gy, int gx, void* stream) {
    if (!nbr || gz < 1 || gy < 1 || gx < 1) return GAMER_EINVAL;
    const long long n = (long long)gz * gy * gx * 27;
    if (n > 0x7fffffff) return GAMER_EUNSUPPORTED;
    neighbors_periodic_kernel<<<(unsigned)((n + 255) / 256), 256, 0, static_cast<cudaStream_t>(stream)>>>(nbr, gz, gy, gx);
    g_launches += 1;
    return cudaGetLastError() == cudaSuccess ? GAMER_OK : GAMER_ECUDA;
}

// ------------------------------------------------------------------------------------------ CFL
template <typename T>
static int cfl_typed(const void* u, int64_t n_groups, double dh, double gamma, double cfl, int scheme,
                     void* group_speed_out, double* dt_out, const gamer_opts* o) {
    cudaStream_t st = o ? static_cast<cudaStream_t>(o->stream) : nullptr;
    CflArgs<T> a;
    a.u = static_cast<const T*>(u);
    a.speed = static_cast<T*>(group_speed_out);
    a.acc = dt_out;
    a.gamma = gamma;
    a.min_dens = o ? o->min_dens : 0.0; a.min_pres = o ? o->min_pres : 0.0; a.min_temp = o ? o->min_temp : 0.0;
    a.n_groups = n_groups;
    a.nvar = 5 + (o ? o->n_scalar : 0);
    if (cudaMemsetAsync(dt_out, 0, sizeof(double), st) != cudaSuccess) return GAMER_ECUDA;
    if (n_groups > 0) {
        const unsigned grid = (unsigned)n_groups;
        if (scheme != GAMER_CTU) {      // Eq. (2): MHM and VL (L168)
            cfl_kernel<T, MHM><<<grid, 256, 0, st>>>(a);
        } else {
            cfl_kernel<T, CTU><<<grid, 256, 0, st>>>(a);
        }
        g_launches += 1;
    }
    finish_dt_kernel<<<1, 1, 0, st>>>(dt_out, cfl * dh);
    g_launches += 1;
    return cudaGetLastError() == cudaSuccess ? GAMER_OK : GAMER_ECUDA;
}

extern "C" int gamer_cfl_dt_ex(const void* u, int64_t n_groups, double dh, double gamma, double cfl, int scheme,
                               int precision, void* group_speed_out, double* dt_out, const gamer_opts* opts) {
    if (!u || !dt_out || n_groups < 0 || !(dh > 0.0) || !(gamma > 1.0) || !(cfl > 0.0)) return GAMER_EINVAL;
    if (scheme != GAMER_MHM && scheme != GAMER_CTU && scheme != GAMER_VL) return GAMER_EINVAL;
    if (precision != GAMER_FP32 && precision != GAMER_FP64) return GAMER_EINVAL;
    if (!aligned16(u)) return GAMER_EINVAL;
    if (opts && (opts->n_scalar < 0 || opts->n_scalar > GAMER_MAX_SCALARS)) return GAMER_EINVAL;
    if (n_groups > 0x7fffffff) return GAMER_EUNSUPPORTED;
    return precision == GAMER_FP32 ? cfl_typed<float>(u, n_groups, dh, gamma, cfl, scheme, group_speed_out, dt_out, opts)
                                   : cfl_typed<double>(u, n_groups, dh, gamma, cfl, scheme, group_speed_out, dt_out, opts);
}

extern "C" int gamer_cfl_dt(const void* u, int64_t n_groups, double dh, double gamma, double cfl, int scheme,
                            int precision, void* group_speed_out, double* dt_out) {
    return gamer_cfl_dt_ex(u, n_groups, dh, gamma, cfl, scheme, precision, group_speed_out, dt_out, nullptr);
}

extern "C" int gamer_cfl_from_group_speed(const void* group_speed, int64_t n_groups, double dh, double cfl,
                                          int precision, double* dt_out, void* stream) {
    if (!group_speed || !dt_out || n_groups < 0 || !(dh > 0.0) || !(cfl > 0.0)) return GAMER_EINVAL;
    if (precision != GAMER_FP32 && precision != GAMER_FP64) return GAMER_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (cudaMemsetAsync(dt_out, 0, sizeof(double), st) != cudaSuccess) return GAMER_ECUDA;
    if (n_groups > 0) {
        const unsigned grid = (unsigned)((n_groups + 8191) / 8192 > 64 ? 64 : (n_groups + 8191) / 8192);
        if (precision == GAMER_FP32)
            group_max_kernel<float><<<grid, 1024, 0, st>>>(static_cast<const float*>(group_speed), n_groups, dt_out);
        else
            group_max_kernel<double><<<grid, 1024, 0, st>>>(static_cast<const double*>(group_speed), n_groups, dt_out);
        g_launches += 1;
    }
    finish_dt_kernel<<<1, 1, 0, st>>>(dt_out, cfl * dh);
    g_launches += 1;
    return cudaGetLastError() == cudaSuccess ? GAMER_OK : GAMER_ECUDA;
}

// ------------------------------------------------------------------------------------------ ghost refresh
extern "C" int gamer_refresh_ghosts_periodic(const void* u, void* in, int gz, int gy, int gx, int nvar, int precision,
                                             void* stream) {
    if (!u || !in || gz < 1 || gy < 1 || gx < 1 || nvar < 5 || nvar > 5 + GAMER_MAX_SCALARS) return GAMER_EINVAL;
    if (precision != GAMER_FP32 && precision != GAMER_FP64) return GAMER_EINVAL;
    const long long ng = (long long)gz * gy * gx;
    if (ng * nvar > 0x7fffffff) return GAMER_EUNSUPPORTED;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const unsigned grid = (unsigned)(ng * nvar);
    if (precision == GAMER_FP32)
        refresh_periodic_kernel<float><<<grid, 256, 0, st>>>(static_cast<const float*>(u), static_cast<float*>(in), gz, gy, gx, nvar);
    else
        refresh_periodic_kernel<double><<<grid, 256, 0, st>>>(static_cast<const double*>(u), static_cast<double*>(in), gz, gy, gx, nvar);
    g_launches += 1;
    return cudaGetLastError() == cudaSuccess ? GAMER_OK : GAMER_ECUDA;
}

extern "C" int gamer_refresh_ghosts(const void* u, void* in, int gz, int gy, int gx, int nvar, const int* bc,
                                    int precision, void* stream) {
    if (!u || !in || !bc || gz < 1 || gy < 1 || gx < 1 || nvar < 5 || nvar > 5 + GAMER_MAX_SCALARS) return GAMER_EINVAL;
    if (precision != GAMER_FP32 && precision != GAMER_FP64) return GAMER_EINVAL;
    BcSet b;
    for (int i = 0; i < 6; ++i) {
        if (bc[i] < GAMER_BC_PERIODIC || bc[i] > GAMER_BC_REFLECTING) return GAMER_EINVAL;
        b.v[i] = bc[i];
    }
    for (int a = 0; a < 3; ++a)      // a periodic axis is periodic on both faces
        if ((bc[2 * a] == GAMER_BC_PERIODIC) != (bc[2 * a + 1] == GAMER_BC_PERIODIC)) return GAMER_EINVAL;
    const long long ng = (long long)gz * gy * gx;
    if (ng * nvar > 0x7fffffff) return GAMER_EUNSUPPORTED;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const unsigned grid = (unsigned)(ng * nvar);
    if (precision == GAMER_FP32)
        refresh_bc_kernel<float><<<grid, 256, 0, st>>>(static_cast<const float*>(u), static_cast<float*>(in), gz, gy, gx, nvar, b);
    else
        refresh_bc_kernel<double><<<grid, 256, 0, st>>>(static_cast<const double*>(u), static_cast<double*>(in), gz, gy, gx, nvar, b);
    g_launches += 1;
    return cudaGetLastError() == cudaSuccess ? GAMER_OK : GAMER_ECUDA;
}

extern "C" int gamer_refresh_ghosts_table(const void* u, void* in, const int32_t* nbr, int64_t n_groups, int nvar,
                                          int precision, void* stream) {
    if (n_groups < 0 || nvar < 5 || nvar > 5 + GAMER_MAX_SCALARS || (precision != GAMER_FP32 && precision != GAMER_FP64)) return GAMER_EINVAL;
    if (n_groups > 0 && (!u || !in || !nbr)) return GAMER_EINVAL;
    if (n_groups == 0) return GAMER_OK;
    if (n_groups * nvar > 0x7fffffff) return GAMER_EUNSUPPORTED;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const unsigned grid = (unsigned)(n_groups * nvar);
    if (precision == GAMER_FP32) refresh_table_kernel<float><<<grid, 256, 0, st>>>(static_cast<const float*>(u), static_cast<float*>(in), nbr, nvar);
    else refresh_table_kernel<double><<<grid, 256, 0, st>>>(static_cast<const double*>(u), static_cast<double*>(in), nbr, nvar);
    g_launches += 1;
    return cudaGetLastError() == cudaSuccess ? GAMER_OK : GAMER_ECUDA;
}

// ------------------------------------------------------------------------------------------ coarse-fine fix-up
template <typename T>
static void launch_interp(const void* c0, const void* c1, double w, void* fine, const int32_t* parent, const int32_t* nbr,
                          unsigned grid, int nvar, int monotonic, cudaStream_t st) {
    const T* a0 = static_cast<const T*>(c0);
    const T* a1 = static_cast<const T*>(c1);
    T* f = static_cast<T*>(fine);
    const T w0 = T(1.0 - w), w1 = T(w);
    if (a1) {
        if (monotonic) interpolate_ghosts_kernel<T, true, true><<<grid, INTERP_NT, 0, st>>>(a0, a1, w0, w1, f, parent, nbr, nvar);
        else interpolate_ghosts_kernel<T, true, false><<<grid, INTERP_NT, 0, st>>>(a0, a1, w0, w1, f, parent, nbr, nvar);
    } else {
        if (monotonic) interpolate_ghosts_kernel<T, false, true><<<grid, INTERP_NT, 0, st>>>(a0, a1, w0, w1, f, parent, nbr, nvar);
        else interpolate_ghosts_kernel<T, false, false><<<grid, INTERP_NT, 0, st>>>(a0, a1, w0, w1, f, parent, nbr, nvar);
    }
}

extern "C" int gamer_interpolate_ghosts(const void* coarse_in, const void* coarse_in_new, double w, void* fine_in,
                                        const int32_t* parent, const int32_t* nbr, int64_t n_fine, int nvar,
                                        int monotonic, int precision, void* stream) {
    if (n_fine < 0 || nvar < 1 || nvar > 5 + GAMER_MAX_SCALARS || (precision != GAMER_FP32 && precision != GAMER_FP64)) return GAMER_EINVAL;
    if (coarse_in_new && (!std::isfinite(w) || w < 0.0 || w > 1.0)) return GAMER_EINVAL;
    if (n_fine > 0 && (!coarse_in || !fine_in || !parent || !nbr || coarse_in == fine_in)) return GAMER_EINVAL;
    if (n_fine == 0) return GAMER_OK;
    if (n_fine * nvar > 0x7fffffff) return GAMER_EUNSUPPORTED;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const unsigned grid = (unsigned)(n_fine * nvar);
    if (precision == GAMER_FP32) launch_interp<float>(coarse_in, coarse_in_new, w, fine_in, parent, nbr, grid, nvar, monotonic, st);
    else launch_interp<double>(coarse_in, coarse_in_new, w, fine_in, parent, nbr, grid, nvar, monotonic, st);
    g_launches += 1;
    return cudaGetLastError() == cudaSuccess ? GAMER_OK : GAMER_ECUDA;
}

static int poisson_sor_impl(void* phi, const void* rho, void* acc, void* resid_out, void* flu, int nvar, double dt,
                            int64_t n_patches, double dh, double coeff, double omega, int n_iter, int precision, void* stream) {
    if (n_patches < 0 || n_iter < 0 || (precision != GAMER_FP32 && precision != GAMER_FP64)) return GAMER_EINVAL;
    if (!(dh > 0.0) || !std::isfinite(dh) || !std::isfinite(coeff) || !(omega > 0.0) || !(omega < 2.0)) return GAMER_EINVAL;
    if (n_patches > 0 && (!phi || !rho || !aligned16(phi) || !aligned16(rho))) return GAMER_EINVAL;
    if (flu && (nvar < 5 || nvar > 5 + GAMER_MAX_SCALARS || !std::isfinite(dt) || (n_patches & 7) != 0)) return GAMER_EINVAL;
    if (n_patches == 0) return GAMER_OK;
    if (n_patches > 0x7fffffff) return GAMER_EUNSUPPORTED;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const unsigned grid = (unsigned)n_patches;
    const double ss = coeff * dh * dh, w6 = omega / 6.0, i2 = 1.0 / (2.0 * dh);
    if (precision == GAMER_FP64 &&      // 49.2 KB of dynamic shared memory: above the default limit
        cudaFuncSetAttribute(poisson_sor_kernel<double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SorGeo<double>::BYTES) != cudaSuccess)
        return GAMER_ECUDA;
    if (precision == GAMER_FP32)
        poisson_sor_kernel<float><<<grid, 256, SorGeo<float>::BYTES, st>>>(static_cast<float*>(phi), static_cast<const float*>(rho),
                                                        static_cast<float*>(acc), static_cast<float*>(resid_out), (float)ss, (float)w6,
                                                        (float)i2, n_iter, static_cast<float*>(flu), nvar, (float)dt);
    else
        poisson_sor_kernel<double><<<grid, 256, SorGeo<double>::BYTES, st>>>(static_cast<double*>(phi), static_cast<const double*>(rho),
                                                         static_cast<double*>(acc), static_cast<double*>(resid_out), ss, w6, i2, n_iter,
                                                         static_cast<double*>(flu), nvar, dt);
    g_launches += 1;
    return cudaGetLastError() == cudaSuccess ? GAMER_OK : GAMER_ECUDA;
}

extern "C" int gamer_poisson_sor(void* phi, const void* rho, void* acc, void* resid_out, int64_t n_patches, double dh,
                                 double coeff, double omega, int n_iter, int precision, void* stream) {
    return poisson_sor_impl(phi, rho, acc, resid_out, nullptr, 0, 0.0, n_patches, dh, coeff, omega, n_iter, precision, stream);
}

extern "C" int gamer_poisson_sor_gravity(void* phi, const void* rho, void* acc, void* resid_out, void* flu, int nvar, double dt,
                                         int64_t n_patches, double dh, double coeff, double omega, int n_iter, int precision,
                                         void* stream) {
    if (n_patches > 0 && !flu) return GAMER_EINVAL;
    return poisson_sor_impl(phi, rho, acc, resid_out, flu, nvar, dt, n_patches, dh, coeff, omega, n_iter, precision, stream);
}

extern "C" int gamer_gravity_update(void* flu, const void* acc, int64_t n_patches, int nvar, double dt, int precision, void* stream) {
    if (n_patches < 0 || (n_patches & 7) != 0 || nvar < 5 || nvar > 5 + GAMER_MAX_SCALARS || !std::isfinite(dt)) return GAMER_EINVAL;
    if (precision != GAMER_FP32 && precision != GAMER_FP64) return GAMER_EINVAL;
    if (n_patches > 0 && (!flu || !acc)) return GAMER_EINVAL;
    if (n_patches == 0) return GAMER_OK;
    if (n_patches > 0x7fffffff) return GAMER_EUNSUPPORTED;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (precision == GAMER_FP32)
        gravity_update_kernel<float><<<(unsigned)n_patches, 256, 0, st>>>(static_cast<float*>(flu), static_cast<const float*>(acc), nvar, (float)dt);
    else
        gravity_update_kernel<double><<<(unsigned)n_patches, 256, 0, st>>>(static_cast<double*>(flu), static_cast<const double*>(acc), nvar, dt);
    g_launches += 1;
    return cudaGetLastError() == cudaSuccess ? GAMER_OK : GAMER_ECUDA;
}

extern "C" int gamer_restrict(const void* fine, void* coarse, const int32_t* parent, int64_t n_fine, int nvar,
                              int precision, void* stream) {
    if (n_fine < 0 || nvar < 1 || nvar > 5 + GAMER_MAX_SCALARS || (precision != GAMER_FP32 && precision != GAMER_FP64)) return GAMER_EINVAL;
    if (n_fine > 0 && (!fine || !coarse || !parent)) return GAMER_EINVAL;
    if (n_fine == 0) return GAMER_OK;
    if (n_fine * nvar > 0x7fffffff) return GAMER_EUNSUPPORTED;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const unsigned grid = (unsigned)(n_fine * nvar);
    if (precision == GAMER_FP32) restrict_kernel<float><<<grid, 512, 0, st>>>(static_cast<const float*>(fine), static_cast<float*>(coarse), parent, nvar);
    else restrict_kernel<double><<<grid, 512, 0, st>>>(static_cast<const double*>(fine), static_cast<double*>(coarse), parent, nvar);
    g_launches += 1;
    return cudaGetLastError() == cudaSuccess ? GAMER_OK : GAMER_ECUDA;
}

extern "C" int gamer_flux_accumulate(void* acc, const void* flux, double weight, int64_t n_groups, int nvar, int init,
                                     int precision, void* stream) {
    if (n_groups < 0 || nvar < 1 || nvar > 5 + GAMER_MAX_SCALARS || (precision != GAMER_FP32 && precision != GAMER_FP64)) return GAMER_EINVAL;
    if (n_groups > 0 && (!acc || !flux)) return GAMER_EINVAL;
    if (!std::isfinite(weight)) return GAMER_EINVAL;
    if (n_groups == 0) return GAMER_OK;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const long long n = (long long)n_groups * 9 * nvar * PS * PS;
    const unsigned grid = (unsigned)((n + 1023) / 1024 > 148 * 8 ? 148 * 8 : (n + 1023) / 1024);
    if (precision == GAMER_FP32) flux_accumulate_kernel<float><<<grid, 256, 0, st>>>(static_cast<float*>(acc), static_cast<const float*>(flux), (float)weight, n, init);
    else flux_accumulate_kernel<double><<<grid, 256, 0, st>>>(static_cast<double*>(acc), static_cast<const double*>(flux), weight, n, init);
    g_launches += 1;
    return cudaGetLastError() == cudaSuccess ? GAMER_OK : GAMER_ECUDA;
}

extern "C" int gamer_flux_correct(void* coarse, const void* coarse_flux, const void* fine_flux_avg, const int32_t* table,
                                  int64_t n_entries, int nvar, double lam, int precision, void* stream) {
    if (n_entries < 0 || nvar < 1 || nvar > 5 + GAMER_MAX_SCALARS || (precision != GAMER_FP32 && precision != GAMER_FP64)) return GAMER_EINVAL;
    if (n_entries > 0 && (!coarse || !coarse_flux || !fine_flux_avg || !table)) return GAMER_EINVAL;
    if (!std::isfinite(lam)) return GAMER_EINVAL;
    if (n_entries == 0) return GAMER_OK;
    if (n_entries > 0x7fffffff) return GAMER_EUNSUPPORTED;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    for (int pass = 0; pass < 6; ++pass) {
        if (precision == GAMER_FP32)
            flux_correct_kernel<float><<<(unsigned)n_entries, 64, 0, st>>>(static_cast<float*>(coarse), static_cast<const float*>(coarse_flux),
                                                                          static_cast<const float*>(fine_flux_avg), table, nvar, (float)lam, pass);
        else
            flux_correct_kernel<double><<<(unsigned)n_entries, 64, 0, st>>>(static_cast<double*>(coarse), static_cast<const double*>(coarse_flux),
                                                                           static_cast<const double*>(fine_flux_avg), table, nvar, lam, pass);
        g_launches += 1;
    }
    return cudaGetLastError() == cudaSuccess ? GAMER_OK : GAMER_ECUDA;
}

// ------------------------------------------------------------------------------------------ host-buffer entry
// scratch of the host entry (3 streams, 3 sets of device buffers), kept between calls: allocating and freeing
// ~0.6 GB per call cost more than the copies of a small batch.  Freed by gamer_release_scratch() or at exit.
static void gamer_release_resident_scratch();
static int check_host_opts(const gamer_opts* opts);
namespace {
struct HostScratch {
    static constexpr int NBUF = 3;
    cudaStream_t st[NBUF] = {nullptr, nullptr, nullptr};
    char* d_in[NBUF] = {};
    char* d_out[NBUF] = {};
    char* d_fl[NBUF] = {};
    char* d_sp[NBUF] = {};
    size_t cap_in = 0, cap_out = 0, cap_fl = 0, cap_sp = 0;
    int device = -1;
    std::mutex mu;
    void release() {
        for (int b = 0; b < NBUF; ++b) {
            if (d_in[b]) cudaFree(d_in[b]);
            if (d_out[b]) cudaFree(d_out[b]);
            if (d_fl[b]) cudaFree(d_fl[b]);
            if (d_sp[b]) cudaFree(d_sp[b]);
            if (st[b]) cudaStreamDestroy(st[b]);
            d_in[b] = d_out[b] = d_fl[b] = d_sp[b] = nullptr;
            st[b] = nullptr;
        }
        cap_in = cap_out = cap_fl = cap_sp = 0;
        device = -1;
    }
    bool ensure(size_t in_b, size_t out_b, size_t fl_b, size_t sp_b) {
        int dev = 0;
        if (cudaGetDevice(&dev) != cudaSuccess) return false;
        if (dev != device || in_b > cap_in || out_b > cap_out || fl_b > cap_fl || sp_b > cap_sp) {
            release();
            for (int b = 0; b < NBUF; ++b) {
                if (cudaStreamCreateWithFlags(&st[b], cudaStreamNonBlocking) != cudaSuccess) return false;
                if (cudaMalloc(&d_in[b], in_b) != cudaSuccess || cudaMalloc(&d_out[b], out_b) != cudaSuccess ||
                    cudaMalloc(&d_fl[b], fl_b) != cudaSuccess || cudaMalloc(&d_sp[b], sp_b) != cudaSuccess)
                    return false;
            }
            cap_in = in_b; cap_out = out_b; cap_fl = fl_b; cap_sp = sp_b;
            device = dev;
        }
        return true;
    }
};
HostScratch g_scratch;
}  // namespace

extern "C" void gamer_release_scratch(void) {
    {
        std::lock_guard<std::mutex> lock(g_scratch.mu);
        g_scratch.release();
    }
    gamer_release_resident_scratch();
}

extern "C" int gamer_fluid_advance_host(const void* in_host, void* out_host, void* flux_out_host,
                                        void* group_speed_out_host, int64_t n_groups, double dt, double dh,
                                        double gamma, int scheme, int recon, int riemann, int precision,
                                        const gamer_opts* opts) {
    if (!in_host || !out_host || n_groups < 0) return GAMER_EINVAL;
    if (precision != GAMER_FP32 && precision != GAMER_FP64) return GAMER_EINVAL;
    if (!(dt > 0.0) || !std::isfinite(dt)) return GAMER_EINVAL;
    {
        const int vrc = check_host_opts(opts);      // before anything is sized from opts
        if (vrc) return vrc;
    }
    if (n_groups == 0) return GAMER_OK;
    const int nv = 5 + (opts ? opts->n_scalar : 0);
    const size_t sz = (size_t)precision;
    const size_t in_g = (size_t)nv * NPC * sz, out_g = (size_t)nv * PS * PS * PS * sz, fl_g = (size_t)9 * nv * PS * PS * sz;
    constexpr int NBUF = HostScratch::NBUF;
    const int64_t chunk = n_groups < 592 ? n_groups : 592;   // 2 waves of 296 CTAs; ~1e6 cells saturate (L321)
    std::lock_guard<std::mutex> lock(g_scratch.mu);
    if (!g_scratch.ensure(in_g * chunk, out_g * chunk, fl_g * chunk, sz * chunk)) {
        g_scratch.release();
        return GAMER_ECUDA;
    }
    cudaStream_t* st = g_scratch.st;
    char **d_in = g_scratch.d_in, **d_out = g_scratch.d_out, **d_fl = g_scratch.d_fl, **d_sp = g_scratch.d_sp;
    int rc = GAMER_OK;
    int64_t done = 0;
    for (int it = 0; done < n_groups && rc == GAMER_OK; ++it) {
        const int b = it % NBUF;
        const int64_t n = (n_groups - done) < chunk ? (n_groups - done) : chunk;
        gamer_opts o;
        if (opts) o = *opts; else std::memset(&o, 0, sizeof(o));
        o.stream = st[b];
        o.dt_dev = nullptr; o.n_unphysical_out = nullptr; o.diag_out = nullptr;
        o.group_speed_out = group_speed_out_host ? d_sp[b] : nullptr;
        const char* hin = static_cast<const char*>(in_host) + done * in_g;
        if (cudaMemcpyAsync(d_in[b], hin, in_g * n, cudaMemcpyHostToDevice, st[b]) != cudaSuccess) { rc = GAMER_ECUDA; break; }
        rc = gamer_fluid_advance_ex(d_in[b], d_out[b], flux_out_host ? d_fl[b] : nullptr, n, dt, dh, gamma, scheme, recon,
                                    riemann, precision, &o);
        if (rc != GAMER_OK) break;
        cudaMemcpyAsync(static_cast<char*>(out_host) + done * out_g, d_out[b], out_g * n, cudaMemcpyDeviceToHost, st[b]);
        if (flux_out_host)
            cudaMemcpyAsync(static_cast<char*>(flux_out_host) + done * fl_g, d_fl[b], fl_g * n, cudaMemcpyDeviceToHost, st[b]);
        if (group_speed_out_host)
            cudaMemcpyAsync(static_cast<char*>(group_speed_out_host) + done * sz, d_sp[b], sz * n, cudaMemcpyDeviceToHost, st[b]);
        if (cudaGetLastError() != cudaSuccess) rc = GAMER_ECUDA;
        done += n;
    }
    for (int b = 0; b < NBUF; ++b)
        if (cudaStreamSynchronize(st[b]) != cudaSuccess) rc = GAMER_ECUDA;
    return rc;
}

// ------------------------------------------------------------------------------------------ host entry, unpadded state
// Validation shared by the two host entries: everything that sizes an allocation or a copy is checked BEFORE it is used.
static int check_host_opts(const gamer_opts* opts) {
    if (!opts) return GAMER_OK;
    if (opts->n_scalar < 0 || opts->n_scalar > GAMER_MAX_SCALARS) return GAMER_EINVAL;
    if (opts->dual_energy && opts->n_scalar < 1) return GAMER_EINVAL;
    if (opts->limiter < 0 || opts->limiter > GAMER_LIMITER_VANALBADA) return GAMER_EINVAL;
    if (opts->minmod_theta > 0.0 && !(opts->minmod_theta >= 1.0 && opts->minmod_theta <= 2.0)) return GAMER_EINVAL;
    if (opts->min_dens < 0 || opts->min_pres < 0 || opts->min_temp < 0) return GAMER_EINVAL;
    if (opts->n_unphysical_out || opts->diag_out || opts->dt_dev) return GAMER_EUNSUPPORTED;   // device outputs: use the device entries
    return GAMER_OK;
}

namespace {
struct ResidentScratch {      // device copy of the whole unpadded state + table, and a ring of output chunks
    static constexpr int NBUF = 3;
    cudaStream_t st_in = nullptr, st[NBUF] = {nullptr, nullptr, nullptr};
    char* d_u = nullptr;
    int32_t* d_nbr = nullptr;
    char* d_out[NBUF] = {};
    char* d_fl[NBUF] = {};
    char* d_sp[NBUF] = {};
    std::vector<cudaEvent_t> ev;      // one per input chunk
    size_t cap_u = 0, cap_nbr = 0, cap_out = 0, cap_fl = 0, cap_sp = 0;
    int device = -1;
    std::mutex mu;
    void release() {
        if (d_u) cudaFree(d_u);
        if (d_nbr) cudaFree(d_nbr);
        for (int b = 0; b < NBUF; ++b) {
            if (d_out[b]) cudaFree(d_out[b]);
            if (d_fl[b]) cudaFree(d_fl[b]);
            if (d_sp[b]) cudaFree(d_sp[b]);
            if (st[b]) cudaStreamDestroy(st[b]);
            d_out[b] = d_fl[b] = d_sp[b] = nullptr;
            st[b] = nullptr;
        }
        if (st_in) cudaStreamDestroy(st_in);
        for (cudaEvent_t e : ev) cudaEventDestroy(e);
        ev.clear();
        d_u = nullptr; d_nbr = nullptr; st_in = nullptr;
        cap_u = cap_nbr = cap_out = cap_fl = cap_sp = 0;
        device = -1;
    }
    bool ensure(size_t u_b, size_t nbr_b, size_t out_b, size_t fl_b, size_t sp_b, size_t n_ev) {
        int dev = 0;
        if (cudaGetDevice(&dev) != cudaSuccess) return false;
        if (dev != device || u_b > cap_u || nbr_b > cap_nbr || out_b > cap_out || fl_b > cap_fl || sp_b > cap_sp) {
            release();
            if (cudaStreamCreateWithFlags(&st_in, cudaStreamNonBlocking) != cudaSuccess) return false;
            if (cudaMalloc(&d_u, u_b) != cudaSuccess || cudaMalloc(&d_nbr, nbr_b) != cudaSuccess) return false;
            for (int b = 0; b < NBUF; ++b) {
                if (cudaStreamCreateWithFlags(&st[b], cudaStreamNonBlocking) != cudaSuccess) return false;
                if (cudaMalloc(&d_out[b], out_b) != cudaSuccess || cudaMalloc(&d_fl[b], fl_b) != cudaSuccess ||
                    cudaMalloc(&d_sp[b], sp_b) != cudaSuccess)
                    return false;
            }
            cap_u = u_b; cap_nbr = nbr_b; cap_out = out_b; cap_fl = fl_b; cap_sp = sp_b;
            device = dev;
        }
        while (ev.size() < n_ev) {
            cudaEvent_t e;
            if (cudaEventCreateWithFlags(&e, cudaEventDisableTiming) != cudaSuccess) return false;
            ev.push_back(e);
        }
        return true;
    }
};
ResidentScratch g_resident;
}  // namespace

extern "C" int gamer_fluid_advance_host_resident(const void* u_host, const int32_t* nbr_host, void* out_host,
                                                 void* flux_out_host, void* group_speed_out_host, int64_t n_groups,
                                                 double dt, double dh, double gamma, int scheme, int recon, int riemann,
                                                 int precision, const gamer_opts* opts) {
    if (!u_host || !nbr_host || !out_host || n_groups < 0 || u_host == out_host) return GAMER_EINVAL;
    if (precision != GAMER_FP32 && precision != GAMER_FP64) return GAMER_EINVAL;
    if (!(dt > 0.0) || !std::isfinite(dt)) return GAMER_EINVAL;
    int rc = check_host_opts(opts);
    if (rc) return rc;
    if (opts && opts->remedy_first_order) return GAMER_EUNSUPPORTED;      // remedy (ii) re-reads the padded slab
    if (n_groups > 0x3fffffff / 27) return GAMER_EUNSUPPORTED;
    if (n_groups == 0) return GAMER_OK;
    const int nv = 5 + (opts ? opts->n_scalar : 0);
    const size_t sz = (size_t)precision;
    const size_t u_g = (size_t)nv * PS * PS * PS * sz, fl_g = (size_t)9 * nv * PS * PS * sz;
    const int64_t chunk = n_groups < 1024 ? n_groups : 1024;      // input and output granularity
    const int64_t n_chunks = (n_groups + chunk - 1) / chunk;
    constexpr int NBUF = ResidentScratch::NBUF;
    std::lock_guard<std::mutex> lock(g_resident.mu);
    ResidentScratch& R = g_resident;
    if (!R.ensure(u_g * n_groups, sizeof(int32_t) * 27 * n_groups, u_g * chunk, fl_g * chunk, sz * chunk, (size_t)n_chunks)) {
        R.release();
        return GAMER_ECUDA;
    }
    // the whole unpadded state goes to the device once, chunk by chunk on its own stream; the table first
    if (cudaMemcpyAsync(R.d_nbr, nbr_host, sizeof(int32_t) * 27 * n_groups, cudaMemcpyHostToDevice, R.st_in) != cudaSuccess) return GAMER_ECUDA;
    for (int64_t k = 0; k < n_chunks; ++k) {
        const int64_t g0 = k * chunk, n = (n_groups - g0) < chunk ? (n_groups - g0) : chunk;
        if (cudaMemcpyAsync(R.d_u + g0 * u_g, static_cast<const char*>(u_host) + g0 * u_g, u_g * n, cudaMemcpyHostToDevice, R.st_in) != cudaSuccess ||
            cudaEventRecord(R.ev[(size_t)k], R.st_in) != cudaSuccess)
            return GAMER_ECUDA;
    }
    // which input chunks each output chunk needs: those that hold one of its groups' 27 table entries.  Walked while the
    // copies above are in flight (885k entries for 32,768 groups: milliseconds of host time); a bad entry is reported after
    // the streams have drained
    std::vector<std::vector<int>> need((size_t)n_chunks);
    bool bad_entry = false;
    {
        std::vector<char> mark((size_t)n_chunks);
        const uint32_t ng = (uint32_t)n_groups, ch = (uint32_t)chunk;
        for (int64_t k = 0; k < n_chunks; ++k) {
            std::fill(mark.begin(), mark.end(), 0);
            const int64_t g1 = (k + 1) * chunk < n_groups ? (k + 1) * chunk : n_groups;
            for (int64_t i = k * chunk * 27; i < g1 * 27; ++i) {
                const uint32_t sidx = (uint32_t)nbr_host[i];      // a negative entry wraps above n_groups
                if (sidx >= ng) { bad_entry = true; continue; }
                mark[(size_t)(sidx / ch)] = 1;
            }
            for (int64_t c = 0; c < n_chunks; ++c)
                if (mark[(size_t)c]) need[(size_t)k].push_back((int)c);
            if (need[(size_t)k].empty()) need[(size_t)k].push_back((int)k);
        }
    }
    if (bad_entry) {
        cudaStreamSynchronize(R.st_in);
        return GAMER_EINVAL;
    }
    // Output chunks are launched in the order in which their inputs arrive (the last input chunk each needs), not in index
    // order: in a periodic box chunk 0 needs the LAST input chunk, and launched first it would hold its stream -- a third of
    // all output chunks queued behind it -- until the whole state is on the device.
    std::vector<int64_t> order((size_t)n_chunks);
    for (int64_t k = 0; k < n_chunks; ++k) order[(size_t)k] = k;
    std::stable_sort(order.begin(), order.end(), [&](int64_t a, int64_t b) { return need[(size_t)a].back() < need[(size_t)b].back(); });
    rc = GAMER_OK;
    for (int64_t pos = 0; pos < n_chunks && rc == GAMER_OK; ++pos) {
        const int64_t k = order[(size_t)pos];
        const int b = (int)(pos % NBUF);
        const int64_t g0 = k * chunk, n = (n_groups - g0) < chunk ? (n_groups - g0) : chunk;
        for (int c : need[(size_t)k])
            if (cudaStreamWaitEvent(R.st[b], R.ev[(size_t)c], 0) != cudaSuccess) rc = GAMER_ECUDA;
        if (rc != GAMER_OK) break;
        gamer_opts o;
        if (opts) o = *opts; else std::memset(&o, 0, sizeof(o));
        o.stream = R.st[b];
        o.dt_dev = nullptr; o.n_unphysical_out = nullptr; o.diag_out = nullptr;
        o.group_speed_out = group_speed_out_host ? R.d_sp[b] : nullptr;
        // the kernel indexes `in` by the table's (global) entries and out / flux / speed by the group's index in the launch
        rc = precision == GAMER_FP32
                 ? advance_typed<float>(R.d_u, R.d_out[b], flux_out_host ? R.d_fl[b] : nullptr, n, dt, dh, gamma, scheme, recon, riemann, &o, R.d_nbr + g0 * 27)
                 : advance_typed<double>(R.d_u, R.d_out[b], flux_out_host ? R.d_fl[b] : nullptr, n, dt, dh, gamma, scheme, recon, riemann, &o, R.d_nbr + g0 * 27);
        if (rc != GAMER_OK) break;
        cudaMemcpyAsync(static_cast<char*>(out_host) + g0 * u_g, R.d_out[b], u_g * n, cudaMemcpyDeviceToHost, R.st[b]);
        if (flux_out_host)
            cudaMemcpyAsync(static_cast<char*>(flux_out_host) + g0 * fl_g, R.d_fl[b], fl_g * n, cudaMemcpyDeviceToHost, R.st[b]);
        if (group_speed_out_host)
            cudaMemcpyAsync(static_cast<char*>(group_speed_out_host) + g0 * sz, R.d_sp[b], sz * n, cudaMemcpyDeviceToHost, R.st[b]);
        if (cudaGetLastError() != cudaSuccess) rc = GAMER_ECUDA;
    }
    if (cudaStreamSynchronize(R.st_in) != cudaSuccess) rc = GAMER_ECUDA;
    for (int b = 0; b < NBUF; ++b)
        if (cudaStreamSynchronize(R.st[b]) != cudaSuccess) rc = GAMER_ECUDA;
    return rc;
}

static void gamer_release_resident_scratch() {
    std::lock_guard<std::mutex> lock(g_resident.mu);
    g_resident.release();
}

extern "C" int64_t gamer_launch_count(void) { return g_launches.load(); }

extern "C" const char* gamer_strerror(int code) {
    switch (code) {
    case GAMER_OK: return "success";
    case GAMER_EINVAL: return "invalid argument";
    case GAMER_EUNSUPPORTED: return "unsupported combination or size";
    case GAMER_ECUDA: return "CUDA runtime or launch error";
    case GAMER_EUNPHYSICAL: return "unphysical cells remain at the minimum time-step";
    case GAMER_ETOOLARGE: return "batch exceeds the static scratch array of the allocation-free entry";
    default: return "unknown error code";
    }
}

extern "C" int gamer_version(void) { return 100; }
