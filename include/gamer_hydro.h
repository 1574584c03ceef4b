/*
 * gamer_hydro.h -- C ABI of the B200-native batched patch-group hydrodynamic solver
 * (the data-parallel hot path of GAMER-2, arXiv 1712.07070; PAPER.md = the paper's text).
 *
 * One call advances a batch of AMR patch groups (8 sibling patches of 8^3 cells
 * = 16^3 cells), each padded with 3 ghost zones per side (L300), by one step of an unsplit
 * Godunov scheme for the ideal-gas Euler equations (section 2.2): MUSCL-Hancock (MHM)
 * or its VL variant, or corner-transport-upwind (CTU, 6 Riemann solves per cell), PLM or PPM reconstruction on
 * primitive variables, Roe / HLLC / HLLE Riemann solver, conservative update.  It also emits
 * the patch-boundary fluxes the AMR flux fix-up needs (L112) and the per-group CFL maximum
 * (Eqs. 1-2; the paper computes time-steps on the GPU too, L240).
 *
 * All work runs in hand-written sm_100a CUDA kernels; there is no CPU fallback.  Every entry
 * point returns 0 on success or a negative GAMER_E* code, never throws, never aborts, and
 * (except the *_host entry) never synchronises: work is enqueued on the given stream.
 *
 * Layouts (x fastest; real = float or double as selected by `precision`):
 *   in        [n_groups][NVAR][22][22][22]   conserved (rho, mx, my, mz, E [, s]); cell (i,j,k) of
 *                                            the group is padded cell (i+3, j+3, k+3)
 *   out       [n_groups][NVAR][16][16][16]
 *   flux_out  [n_groups][3 axes][3 planes][NVAR][16][16]   plane p of axis d = the cell face at
 *             index 8p of that axis (faces of the 8^3 patches); the two 16-long dims are the two
 *             other axes, the lower-numbered axis fastest (x-faces: [z][y]; y: [z][x]; z: [y][x]).
 *             Values are the time-centred flux densities F_d, not multiplied by dt or area.
 *   group_speed_out [n_groups]   max over the 16^3 UPDATED cells of |vx|+|vy|+|vz|+3c (MHM and VL, Eq. 2)
 *                                or max(|vx|,|vy|,|vz|)+c (CTU, Eq. 1).  A cell whose speed is NaN (P < 0 after the update)
 *                                is skipped by the maximum: such cells are reported through n_unphysical_out, which is what
 *                                a caller must test (remedies (iv)/(v)); the dt of the remaining cells stays usable
 *   NVAR = 5 + n_scalar: conserved passive scalars s_k (chemical species as partial densities, L96) follow E; each
 *   is reconstructed as q_k = s_k / rho and rides the mass flux, upwinded.  With dual_energy the last one carries the
 *   entropy s = P/rho^(gamma-1) of L100.
 * Ownership: every pointer is a DEVICE pointer owned by the caller, 16-byte aligned and
 * non-overlapping, unless the name ends in _host.  The device entries keep no state between calls; the two *_host entries
 * keep their streams and device scratch buffers until gamer_release_scratch() and serialise their callers on a mutex.
 */
#ifndef GAMER_HYDRO_H
#define GAMER_HYDRO_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { GAMER_MHM = 1, GAMER_CTU = 2,
       GAMER_VL = 3 };      /* scheme (L90).  VL = "a variant of the MUSCL-Hancock scheme (VL; Falle 1991; van Leer 2006)":
                               the half-step predictor is a first-order Godunov update of the cell averages (the same Riemann
                               solver on piecewise-constant data), the face values are then reconstructed from that half-step
                               state; 6 Riemann solves per cell; CFL by Eq. (2) like MHM (L168).  PLM only: with PPM the scheme
                               would read a fourth ghost zone, the layout fixes three (L300) -> GAMER_EUNSUPPORTED */
enum { GAMER_PLM = 1, GAMER_PPM = 2 };                      /* recon    (L94)            */
enum { GAMER_ROE = 1, GAMER_HLLC = 2, GAMER_HLLE = 3,
       GAMER_EXACT = 4 };   /* riemann (L94); EXACT = Toro (2009) ch. 4, iterative: Newton on the pressure function
                               from the two-rarefaction guess, vacuum-generating data handled by HLLE */
#define GAMER_MAX_SCALARS 4   /* passive scalars the kernels are built for (the paper: "an arbitrary number", L96) */
enum { GAMER_FP32 = 4, GAMER_FP64 = 8 };                    /* precision = sizeof(real), L244 */
enum { GAMER_LIMITER_GMINMOD = 1, GAMER_LIMITER_VANLEER = 2, GAMER_LIMITER_VANALBADA = 3 }; /* L94 */

enum {
    GAMER_OK = 0,
    GAMER_EINVAL = -1,        /* NULL in/out, n_groups < 0, dt <= 0 or non-finite, dh <= 0, gamma <= 1,
                                 unknown enum, misaligned pointer                                  */
    GAMER_EUNSUPPORTED = -2,  /* valid arguments, combination not built                            */
    GAMER_ECUDA = -3,         /* CUDA runtime / launch error (cudaGetLastError)                    */
    GAMER_EUNPHYSICAL = -4,   /* gamer_fluid_advance_retry only: remedy (v) of L108 gave up at dt_min */
    GAMER_ETOOLARGE = -5      /* gamer_fluid_advance_table_noalloc only: the batch exceeds the static scratch array */
};

/* Everything the 11-argument form fixes by default.  Zero-initialise, then set what you need. */
typedef struct gamer_opts {
    void*    stream;              /* cudaStream_t; NULL = default stream                            */
    int      limiter;             /* GAMER_LIMITER_*; 0 = generalized minmod                        */
    double   minmod_theta;        /* <= 0: 1 for PLM (plain minmod), 2 for PPM (Colella-Woodward); else must lie in [1, 2]
                                     (the TVD range), anything else is GAMER_EINVAL                 */
    int      n_scalar;            /* 0 .. GAMER_MAX_SCALARS passively advected scalars (L96)        */
    int      dual_energy;         /* 0 | 1 (needs n_scalar >= 1; the LAST scalar is the entropy): L100 */
    double   de_xi;               /* switch E_the/E_kin < xi; <= 0: 1e-2                            */
    double   min_dens, min_pres, min_temp;   /* floors, 0 = off; temperature = P/rho (L504)         */
    int      remedy_first_order;  /* 1: remedy (ii) of L105 on cells that come out unphysical       */
    const double* dt_dev;         /* nullable device double: if set, dt is read from it on device   */
    void*    group_speed_out;     /* nullable real[n_groups]                                        */
    int32_t* n_unphysical_out;    /* nullable device int: cells still unphysical after the remedies;
                                     the caller applies remedy (iv) (retry with 0.8 dt, L107)       */
    int32_t* diag_out;            /* nullable device int[4], set by the call: {remedy (i) faces,
                                     reverted predictor states, remedy (ii) cells, dual-energy fixes} */
    int      char_limiting;       /* 1: slopes limited in characteristic variables (L94): R . limiter(L dW-, L dW+)
                                     with the eigenvectors of the cell; 0: in primitive variables (default)    */
    int      renormalize;         /* 1: after every update rescale the passive scalars so that they sum to rho, i.e. the
                                     mass fractions to unity (L96): s_k <- s_k rho / sum_k s_k over all scalars except the
                                     entropy of the dual-energy formalism; a cell whose sum is not positive is left alone   */
} gamer_opts;

/* One step for n_groups patch groups.  flux_out may be NULL.  n_groups == 0 is a successful no-op.
 * Defaults: gen. minmod (theta 1 for PLM, 2 for PPM), primitive-variable reconstruction, no scalar,
 * no dual energy, no floors, remedy (i) (Roe -> HLLE on faces whose intermediate states are
 * unphysical, L104) on, remedy (ii) off. */
int gamer_fluid_advance(const void* in, void* out, void* flux_out, int64_t n_groups,
                        double dt, double dh, double gamma,
                        int scheme, int recon, int riemann, int precision);

int gamer_fluid_advance_ex(const void* in, void* out, void* flux_out, int64_t n_groups,
                           double dt, double dh, double gamma,
                           int scheme, int recon, int riemann, int precision,
                           const gamer_opts* opts);

/* Remedies (iv) and (v) of PAPER.md L107-108 around gamer_fluid_advance_ex: run the step; while the count of cells still
 * unphysical after the in-kernel remedies (i), (ii) and the floors is not zero, "reduce the time-step by a fixed ratio
 * (0.8 by default) and recalculate all patches" -- the whole batch again from the same `in` with dt <- dt * dt_ratio --
 * "until no unphysical results are detected or reaching a given minimum time-step threshold": when the reduced dt falls
 * below dt_min (or after 200 reductions) the call returns GAMER_EUNPHYSICAL, the caller's abort, with `out` holding the
 * last attempt.  opts must be non-NULL with n_unphysical_out set (device int32; holds the last attempt's count on return)
 * and dt_dev NULL; dt_ratio in (0,1), <= 0 = 0.8; dt_min >= 0.  *dt_used_host (nullable, HOST double) = the step of the
 * last attempt = dt multiplied *n_retries_host (nullable, HOST int32) times by dt_ratio.  Unlike the other device entry
 * points this one synchronises opts->stream after every attempt (it reads the count back). */
int gamer_fluid_advance_retry(const void* in, void* out, void* flux_out, int64_t n_groups,
                              double dt, double dh, double gamma,
                              int scheme, int recon, int riemann, int precision,
                              const gamer_opts* opts, double dt_ratio, double dt_min,
                              double* dt_used_host, int32_t* n_retries_host);

/* CFL time-step of an UNPADDED state u (the `out` layout): Eq. (2) for MHM, Eq. (1) for CTU.
 * *dt_out (device double) = cfl * dh / max speed.  group_speed_out nullable.
 * The _ex form takes stream, n_scalar and the floors from opts (others ignored). */
int gamer_cfl_dt(const void* u, int64_t n_groups, double dh, double gamma, double cfl,
                 int scheme, int precision, void* group_speed_out, double* dt_out);
int gamer_cfl_dt_ex(const void* u, int64_t n_groups, double dh, double gamma, double cfl,
                    int scheme, int precision, void* group_speed_out, double* dt_out,
                    const gamer_opts* opts);

/* dt from the per-group maxima that gamer_fluid_advance_ex already produced (fused A8 row):
 * *dt_out = cfl * dh / max_g group_speed[g]. */
int gamer_cfl_from_group_speed(const void* group_speed, int64_t n_groups, double dh, double cfl,
                               int precision, double* dt_out, void* stream);

/* Same-level ghost refresh on the device for a periodic box of gz x gy x gx patch groups
 * (g = (z*gy + y)*gx + x): builds the padded `in` batch from the unpadded `u` batch (the paper's
 * CPU "preparation" step for sibling copies, L248).  u and in must not overlap. */
int gamer_refresh_ghosts_periodic(const void* u, void* in, int gz, int gy, int gx, int nvar,
                                  int precision, void* stream);

/* The same for a uniform level with the standard boundary conditions of PAPER.md L98, set per face:
 * bc[6] = {x_lo, x_hi, y_lo, y_hi, z_lo, z_hi} (host ints), GAMER_BC_PERIODIC (ghost cell c takes cell c mod n),
 * GAMER_BC_OUTFLOW (zero gradient: the nearest cell inside) or GAMER_BC_REFLECTING (the mirror cell -1-c / 2n-1-c
 * with the momentum normal to that face negated).  Inflow (user-defined) boundaries are the caller's own fill. */
#define GAMER_BC_PERIODIC   0
#define GAMER_BC_OUTFLOW    1
#define GAMER_BC_REFLECTING 2
int gamer_refresh_ghosts(const void* u, void* in, int gz, int gy, int gx, int nvar, const int* bc,
                         int precision, void* stream);

/* The sibling copy for any same-level topology: nbr[n_groups][27] (device int32) as in gamer_fluid_advance_resident,
 * except that an entry may be -1 = "no same-level neighbour there" (a coarse-fine or domain boundary): those slabs of
 * `in` are left as they are, for the caller to fill (interpolation from the parent level, user-defined inflow). */
int gamer_refresh_ghosts_table(const void* u, void* in, const int32_t* nbr, int64_t n_groups, int nvar,
                               int precision, void* stream);

/* Ghost zones at coarse-fine boundaries, "interpolating from coarse patches", with the temporal interpolation
 * between the coarse level's two stored times (L482): the companion of gamer_refresh_ghosts_table, it fills exactly the slabs
 * of fine_in[n_fine][nvar][22][22][22] whose entry in nbr[n_fine][27] (the FINE level's same-level table) is negative and
 * touches nothing else.  coarse_in[..][nvar][22][22][22] is the PADDED coarse batch (ghosts filled: the stencil reaches one
 * coarse cell beyond the two that 3 fine ghost cells cover); parent[g] (device int32) = coarse group * 8 + octant
 * (oz*4 + oy*2 + ox) refined by fine group g, as in gamer_restrict.  The paper names no spatial scheme for the fluid; this is
 * conservative piecewise-linear interpolation of the conserved variables (R24):
 *   child = U_c + ((+-s_z) + (+-s_y) + (+-s_x)) / 4,   + for the upper child along that axis,
 *   s_d = (U_{c+e_d} - U_{c-e_d}) / 2 (monotonic = 0) or minmod(U_c - U_{c-e_d}, U_{c+e_d} - U_c) (monotonic = 1),
 * so that the 8 children of a coarse cell average to it.  U = coarse_in, or (1-w) * coarse_in + w * coarse_in_new when
 * coarse_in_new is non-NULL (w in [0,1]: the fine sub-step's time between the two coarse states).  fp64 results are
 * bit-identical to the oracle's loops.  n_fine == 0 is a successful no-op. */
int gamer_interpolate_ghosts(const void* coarse_in, const void* coarse_in_new, double w, void* fine_in,
                             const int32_t* parent, const int32_t* nbr, int64_t n_fine, int nvar,
                             int monotonic, int precision, void* stream);

/* Device-resident step with the same-level ghost refresh FUSED into the staging loads (SURVEY 8(f) NEXT-1,
 * PAPER.md L248 "preparation" + L274 Fig. 3): `u` is the UNPADDED state of the whole batch,
 * u[n_groups][NVAR][16][16][16] (the `out` layout), and nbr[n_groups][27] (device int32) names, for every group,
 * the group that holds each of its 27 same-level neighbours, index (dz+1)*9 + (dy+1)*3 + (dx+1) with
 * d* in {-1,0,+1} (entry 13 = the group itself); every entry must be in [0, n_groups).  The kernel gathers each
 * padded plane from those groups directly, so no padded copy of the batch exists in memory; results are
 * bit-identical to gamer_refresh_ghosts_periodic / a host gather followed by gamer_fluid_advance_ex.
 * u and out must not overlap (every group reads its neighbours' old state).  opts may be NULL.
 * All schemes, reconstructions, solvers and precisions; all opts except remedy_first_order (remedy (ii)
 * re-reads the padded slab), which returns GAMER_EUNSUPPORTED -- use the refresh + gamer_fluid_advance_ex pair there. */
int gamer_fluid_advance_resident(const void* u, const int32_t* nbr, void* out, void* flux_out, int64_t n_groups,
                                 double dt, double dh, double gamma,
                                 int scheme, int recon, int riemann, int precision,
                                 const gamer_opts* opts);

/* Fills nbr[gz*gy*gx][27] (device int32) for a periodic box of gz x gy x gx groups, g = (z*gy + y)*gx + x. */
int gamer_neighbors_periodic(int32_t* nbr, int gz, int gy, int gx, void* stream);

/* ---- The two fix-up operations between a refined level and its parent level,
 * on the same patch-group layouts as the solver.  All pointers are device pointers; nothing is allocated.
 *
 * Restriction: fine[n_fine][nvar][16][16][16] -> the octants of coarse[..][nvar][16][16][16] that the fine groups
 * cover; parent[g] (device int32) = coarse group * 8 + octant, octant = oz*4 + oy*2 + ox.  Each coarse cell becomes
 * 1/8 of the sum of its eight children, added in the order (dz,dy,dx) = (0,0,0), (0,0,1), (0,1,0), ... */
int gamer_restrict(const void* fine, void* coarse, const int32_t* parent, int64_t n_fine, int nvar, int precision,
                   void* stream);

/* acc = (init ? 0 : acc) + weight * flux over n_groups flux_out batches ([n_groups][3][3][nvar][16][16]): the time
 * average of the fine level's flux_out over its sub-steps (weight = dt_sub / dt_coarse). */
int gamer_flux_accumulate(void* acc, const void* flux, double weight, int64_t n_groups, int nvar, int init,
                          int precision, void* stream);

/* Flux correction of the coarse cells next to coarse-fine boundaries:
 *   U_cell += sgn * lam * (avg2x2(fine_flux_avg) - coarse_flux),   lam = dt_coarse / dh_coarse,
 * avg2x2 = 0.25 * (((f00 + f01) + f10) + f11) over the 2 x 2 fine faces of a coarse face.  table[n_entries][8]
 * (device int32), one entry per outer face of a fine group that is a coarse-fine boundary (8 x 8 coarse faces):
 *   [0] fine group  [1] axis d  [2] side: 0 = the group's low face (its flux plane 0, sgn = -1: the face is the upper
 *   face of the corrected cells), 1 = high face (plane 2, sgn = +1)  [3] coarse group whose flux_out holds the coarse
 *   flux of that face  [4] its plane (0,1,2)  [5] (b0 << 8) | a0 = origin of the 8 x 8 quadrant inside that 16 x 16
 *   plane (b = slower, a = faster remaining axis)  [6] coarse group that owns the corrected cells
 *   [7] (z << 16) | (y << 8) | x = the corrected cell with b = a = 0 (its coordinate along d is the cell layer).
 * The entries are applied in six passes (axis 0 side 0, axis 0 side 1, axis 1 side 0, ...); inside a pass no two
 * entries may touch the same cell, so the result does not depend on the execution order (bitwise reproducible). */
int gamer_flux_correct(void* coarse, const void* coarse_flux, const void* fine_flux_avg, const int32_t* table,
                       int64_t n_entries, int nvar, double lam, int precision, void* stream);

/* ---- The paper's other GPU solver: the refined-level Poisson solver of PAPER.md L126-128, L236.
 * Every patch is relaxed independently on its (8 + 2*5)^3 = 18^3 grid (8^3 active zones + 5 buffer zones per side, Fig. 2)
 * "with the outermost cells being fixed during the iterations", 7-point Laplacian, successive over-relaxation in red-black
 * order (R25): n_iter iterations, each = the half-sweep over cells with (i+j+k) even, then odd,
 *   phi += omega / 6 * (sum of the 6 neighbours - 6 phi - coeff * dh^2 * rho),      for laplacian(phi) = coeff * rho.
 * phi[n_patches][18][18][18] (device, in place): initial guess inside (L238: interpolated from the coarse level by the caller)
 * and the boundary condition on the outermost layer, which is returned unchanged; rho[n_patches][16][16][16]: the density on
 * the relaxed cells; acc (nullable) [n_patches][3][8][8][8] = -grad(phi) on the active zones (cells 5..12) by central
 * differences, components (x, y, z) (L238: "the cell-centered gravitational acceleration ... immediately after solving the
 * potential").  resid_out (nullable) real[n_patches] = max over the relaxed cells of |sum of the 6 neighbours - 6 phi -
 * coeff * dh^2 * rho| after the last iteration: dh^2 times the defect of the discretised equation, for the caller to judge "to
 * machine precision" (L126) and iterate on.  0 < omega < 2; n_iter >= 0; the potential lives in shared memory for the whole
 * solve (49.2 KB in fp64). */
int gamer_poisson_sor(void* phi, const void* rho, void* acc, void* resid_out, int64_t n_patches, double dh, double coeff,
                      double omega, int n_iter, int precision, void* stream);

/* The fluid's gravity update, which the paper performs on the GPU "immediately after solving the potential" to save a round
 * trip of the acceleration (L130 "correct momentum and then use the corrected momentum to further correct
 * energy"; R28).  For every cell of the 8^3 active zones of every patch, with g = -grad(phi):
 *   m <- m + dt * rho * g,      E <- E + (|m_new|^2 - |m_old|^2) / (2 rho)      (density, thermal energy and scalars unchanged).
 * flu[n_patches / 8][nvar][16][16][16] is the fluid in the PATCH-GROUP layout (`out` of the solver), updated in place; patch
 * n = 8 g + oz*4 + oy*2 + ox is the octant (ox, oy, oz) of group g (the numbering of gamer_restrict), so n_patches must be a
 * multiple of 8.  gamer_poisson_sor_gravity = gamer_poisson_sor with this update fused behind the solve in the same kernel
 * (the acceleration never leaves the SM; acc may be NULL); gamer_gravity_update applies a given acc[n_patches][3][8][8][8]
 * (e.g. the root level's, or an external acceleration).  A caller builds the second-order corrector of L130 from two
 * half kicks with the old and the new acceleration.  dt may be negative (undoing a kick). */
int gamer_poisson_sor_gravity(void* phi, const void* rho, void* acc, void* resid_out, void* flu, int nvar, double dt,
                              int64_t n_patches, double dh, double coeff, double omega, int n_iter, int precision, void* stream);
int gamer_gravity_update(void* flu, const void* acc, int64_t n_patches, int nvar, double dt, int precision, void* stream);

/* End-to-end form with HOST buffers (pinned or pageable): copies `in` to the device in chunks,
 * runs the solver, copies `out`, `flux_out` (nullable) and `group_speed_out` (nullable) back,
 * overlapping copies and kernels on internal streams as the paper does with CUDA streams (L242),
 * and synchronises before returning.  Three device buffer sets of one chunk (592 groups, about 0.6 GB in fp32) and three
 * streams are created on first use and kept for later calls (gamer_release_scratch frees them); calls are serialised. */
int gamer_fluid_advance_host(const void* in_host, void* out_host, void* flux_out_host,
                             void* group_speed_out_host, int64_t n_groups,
                             double dt, double dh, double gamma,
                             int scheme, int recon, int riemann, int precision,
                             const gamer_opts* opts /* nullable; stream is ignored; n_unphysical_out / diag_out / dt_dev
                                                       set => GAMER_EUNSUPPORTED; invalid fields => GAMER_EINVAL before any copy */);

/* The same from the UNPADDED state: u_host[n_groups][NVAR][16][16][16] and the same-level table nbr_host[n_groups][27]
 * (HOST int32; as in gamer_fluid_advance_resident: entry 13 = the group itself, every entry in [0, n_groups)).  No padded
 * batch exists anywhere: the state crosses PCIe once (1 / 2.6 of the padded bytes), in chunks of 1024 groups on a copy
 * stream; the kernel of output chunk k (gamer_fluid_advance_resident's fused ghost gather, on one of three streams) starts as
 * soon as the input chunks its table entries point into have landed, and its out / flux_out / group_speed_out chunk is copied
 * back behind it -- the paper's preparation step (its stated bottleneck, L681-687) and its stream overlap (L242) without the
 * CPU gather.  The call keeps a device copy of the whole state (n_groups x NVAR x 16 KB in fp32) plus three output chunks
 * between calls (gamer_release_scratch frees them), serialises callers on a mutex and synchronises before returning.
 * fp64 results are bit-identical to gamer_fluid_advance_resident.  Not with remedy_first_order (GAMER_EUNSUPPORTED);
 * opts->n_unphysical_out / diag_out / dt_dev set => GAMER_EUNSUPPORTED (device outputs belong to the device entries).
 * The table is walked on the host while the input copies are already in flight, and output chunks are launched in the order
 * in which their inputs land; a table entry outside [0, n_groups) => GAMER_EINVAL once those copies have drained, with the
 * host outputs untouched. */
int gamer_fluid_advance_host_resident(const void* u_host, const int32_t* nbr_host, void* out_host, void* flux_out_host,
                                      void* group_speed_out_host, int64_t n_groups,
                                      double dt, double dh, double gamma,
                                      int scheme, int recon, int riemann, int precision,
                                      const gamer_opts* opts /* nullable */);

/* Allocation-free step from the UNPADDED state, for callers that cannot call cudaMalloc (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid allocation): u[n_groups][NVAR][16][16][16] and the same-level table nbr[n_groups][27]
 * (device int32, as in gamer_fluid_advance_resident: every entry in [0, n_groups)) in, out / flux_out as everywhere.  The
 * padded batch that gamer_refresh_ghosts_table + gamer_fluid_advance_ex need as caller-allocated scratch lives here in a
 * file-scope static device array of GAMER_NOALLOC_SCRATCH_BYTES (64 MiB; every GPU that loads the library holds it until the
 * process exits): the call runs those same two kernels on it -- results are bit-identical to that pair -- and calls no
 * cudaMalloc, cudaFree or allocating library routine.  Because the padded slab stays in memory, remedy_first_order (remedy
 * (ii), which gamer_fluid_advance_resident cannot offer) works.  All opts as gamer_fluid_advance_ex; work is enqueued on
 * opts->stream, nothing synchronises.
 * Limit: n_groups <= gamer_noalloc_max_groups(NVAR, precision) = 64 MiB / (NVAR * 22^3 * sizeof(real)) -- 315 groups in fp32
 * and 157 in fp64 at NVAR = 5; more returns GAMER_ETOOLARGE and enqueues nothing.
 * ALL CALLS SHARE THE ONE ARRAY per GPU: two calls that overlap on the GPU (different streams, different host threads) race
 * on it; order them on one stream or with events.  The array keeps the last call's contents, so the part a call uses is
 * cleared first: a slab whose table entry is -1 (no same-level neighbour; the allocating path leaves it for the caller's
 * interpolation) is zero here, and cells that depend on it come out non-finite, the same way on every call. */
#define GAMER_NOALLOC_SCRATCH_BYTES (64u << 20)
int gamer_fluid_advance_table_noalloc(const void* u, const int32_t* nbr, void* out, void* flux_out, int64_t n_groups,
                                      double dt, double dh, double gamma,
                                      int scheme, int recon, int riemann, int precision,
                                      const gamer_opts* opts /* nullable */);
int64_t gamer_noalloc_max_groups(int nvar, int precision);

void gamer_release_scratch(void);

/* Measurement helper, not part of the solver (SURVEY 8(d) "ALU peaks to verify on the box"): runs a dependent-free
 * instruction stream of the given kind on every SM (2 x 1024 threads per SM, 8 independent chains per thread), times it with
 * CUDA events on `stream` (best of 5; the call synchronises) and returns the plain-ALU rate it reached:
 * *tflops_out (nullable, HOST double) in TFLOP/s with FMA = 2 FLOPs, *gwarpinst_out (nullable, HOST double) in 1e9 warp
 * instructions per second.  bench.py uses GAMER_ALU_FFMA / GAMER_ALU_DFMA as the measured peaks of the fp32 / fp64 "alu"
 * roofline of the hydro kernels; the mixed streams show how issue slots are shared between the FMA pipe, the ALU pipe
 * (min/max, compares, selects) and the special-function unit.  Allocates and frees 1.2 MB of device scratch. */
enum { GAMER_ALU_FFMA = 0,         /* fp32 FMA, three register operands                                   */
       GAMER_ALU_FMUL_FADD = 1,    /* fp32 multiply and add kept apart: 1 FLOP per issue slot             */
       GAMER_ALU_FFMA_FMNMX = 2,   /* fp32 FMA + min, alternating: FMA pipe + ALU pipe                    */
       GAMER_ALU_FFMA2 = 3,        /* packed fma.rn.f32x2: two FMAs per instruction                       */
       GAMER_ALU_FFMA2_FMNMX = 4,  /* packed FMA + two min                                                */
       GAMER_ALU_DFMA = 5,         /* fp64 FMA                                                            */
       GAMER_ALU_FFMA_MUFU = 6,    /* fp32 FMA with one rcp.approx in every 9 instructions                */
       GAMER_ALU_FFMA2_FFMA = 7,   /* one packed FMA to two plain ones                                    */
       GAMER_ALU_FFMA2_IADD = 8 }; /* packed FMA + integer add, alternating                               */
int gamer_alu_peak(int kind, double* tflops_out, double* gwarpinst_out, void* stream);

/* Number of kernel launches the library has issued in this process (all entry points). */
int64_t gamer_launch_count(void);

const char* gamer_strerror(int code);
int gamer_version(void);

#ifdef __cplusplus
}
#endif
#endif /* GAMER_HYDRO_H */
