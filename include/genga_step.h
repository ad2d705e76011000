/*
 * genga_step.h -- C ABI of the O(N) neighbours of the kick in GENGA's hybrid symplectic step
 * (arXiv 2201.10058, App. A) and of the composed step:
 *
 *     Rcrit(dt)
 *     Kick(dt/2), close-encounter pre-check          <- genga_kick.h
 *     HC(dt/2)
 *     FG(dt)
 *     [ close-encounter detection, grouping, Bulirsch-Stoer: NOT part of this library ]
 *     HC(dt/2)
 *     Kick(dt/2)
 *
 * Every function works on the context of genga_kick.h (its N = n_massive + n_test bodies, its G,
 * its stream), only ENQUEUES kernels on that stream and never synchronises.  All arrays are DEVICE
 * pointers, FP64, 16-byte aligned, owned by the caller; pos and vel are [3][N] SoA in democratic
 * coordinates: heliocentric positions, barycentric velocities.  Units as in
 * genga_kick.h (AU, day, Msun with G = k^2).  There is no CPU fallback.
 *
 * Return codes and genga_kick_strerror as in genga_kick.h.  Device-side conditions are reported
 * through genga_kick_status (GENGA_KICK_STATUS_UNBOUND).
 */
#ifndef GENGA_STEP_H
#define GENGA_STEP_H

#include "genga_kick.h"

#ifdef __cplusplus
extern "C" {
#endif

#define GENGA_KICK_STATUS_UNBOUND 8   /* Rcrit met a body that is not on a bound orbit about the central mass
                                         (1/a = 2/r - v^2/mu <= 0): its Hill term is taken as 0.  FG sets the
                                         bit only for 1/a = 0 exactly (parabolic; the body is left where it is):
                                         a hyperbolic body follows its two-body orbit like any other          */

/*
 * Rcrit: the critical radii of eq. 5, one row per symplectic level (PAPER.md:638:
 * "defined in the same way on each level ... with the reduced time step"):
 *     out_rcrit[k][i] = max(n1 * R_H,i , n2 * (dt / substeps^k) * |v_i|),   k = 0 .. nrows-1
 * with R_H,i = a_i (m_i / (3 m_star))^(1/3), a_i the osculating semi-major axis from the vis-viva
 * equation with mu = G m_star, and |v_i| the speed of the state passed in (reading G6).
 * The paper's constants are n1 = 3, n2 = 0.4.
 * out_rcrit: [nrows][N], the layout genga_kick reads.
 * Errors: E_NULL, E_ALIGN, E_SIZE (nrows < 1, substeps <= 0, m_star <= 0), E_CUDA.
 */
int genga_rcrit(genga_kick_ctx* ctx, const double* pos, const double* vel, const double* mass, double m_star,
                double dt, double substeps, int32_t nrows, double n1, double n2, double* out_rcrit);

/*
 * RcritS / FGS (App. A: "The functions RcritS, KickS, and FGS are similar to the original
 * functions, but are applied only to the relevant bodies in each symplectic level"): genga_rcrit and genga_fg
 * for the bodies of a list only -- e.g. `members` of genga_group.  Bodies not in the list are not read and
 * not written (genga_rcrit_list writes out_rcrit[k][i] for listed i only).  KickS is genga_kick_list.
 *   list      [list_rows] int32 device, 16-byte aligned: body indices, each at most once
 *   n_list    device pointer to ONE int32: number of entries (clipped to list_rows), e.g. summary + 1 of genga_group
 * An index outside [0, N) is ignored and sets status bit 16.
 * Errors: as genga_rcrit / genga_fg, plus E_SIZE for list_rows < 0.
 */
int genga_rcrit_list(genga_kick_ctx* ctx, const double* pos, const double* vel, const double* mass, double m_star,
                     double dt, double substeps, int32_t nrows, double n1, double n2, const int32_t* list,
                     const int32_t* n_list, int64_t list_rows, double* out_rcrit);
int genga_fg_list(genga_kick_ctx* ctx, double* pos, double* vel, double m_star, double dt, const int32_t* list,
                  const int32_t* n_list, int64_t list_rows);

/*
 * HC: the Sun part H_C = (sum_i p_i)^2 / (2 m_star) of eq. 4, "the democratic
 * momentum summation" (App. A): pos_i += dt * (sum_j m_j v_j) / m_star for every
 * body, in place.  The sum runs over all N bodies in a fixed order (bit-reproducible,
 * PAPER.md:1045); velocities are not changed.
 * Errors: E_NULL, E_ALIGN, E_SIZE (m_star <= 0), E_CUDA.
 */
int genga_hc(genga_kick_ctx* ctx, double* pos, const double* vel, const double* mass, double m_star, double dt);

/*
 * FG: the Kepler part of eq. 2: every body advances by dt on its two-body orbit
 * about the central mass, mu = G m_star, with Gauss' f and g functions; pos and vel in place.
 * Elliptic and hyperbolic orbits alike; only a body with 1/a = 0 exactly (parabolic) is left untouched and
 * GENGA_KICK_STATUS_UNBOUND is set.
 * (The pair term [1 - K] of eq. 2 belongs to the Bulirsch-Stoer phase and is not applied here.)
 * Errors: E_NULL, E_ALIGN, E_SIZE (m_star <= 0), E_CUDA.
 */
int genga_fg(genga_kick_ctx* ctx, double* pos, double* vel, double m_star, double dt);

/*
 * HC(dt/2) FG(dt) HC(dt/2) in three launches (momentum sum; shift + Kepler drift + the next
 * momentum sum in one kernel; shift).  Same results as the three calls, bit for bit.
 * Errors: as above.
 */
int genga_drift(genga_kick_ctx* ctx, double* pos, double* vel, const double* mass, double m_star, double dt);

/*
 * One step of the scheme above, without the Bulirsch-Stoer branch:
 *     Rcrit(dt) -> rcrit_row;  Kick(dt/2) + pre-check (level 0);  HC(dt/2);  FG(dt);  HC(dt/2);  Kick(dt/2).
 * pos, vel are advanced in place.  out_pairs / out_npairs receive the close-encounter candidates of
 * the FIRST kick, exactly as genga_kick writes them (the caller's direct solver would act on them
 * after FG; if out_npairs[N] is 0 the step is complete as it stands).  The closing kick writes no
 * pair list.  rcrit_row: [N] scratch/result row, or NULL to use library scratch.  out_acc: [3][N]
 * acceleration of the closing kick, or NULL.
 * The context must have been created with max_level >= 0 (level 0 is used).
 * Errors: E_NULL, E_ALIGN, E_SIZE, E_CUDA.
 */
int genga_step(genga_kick_ctx* ctx, double* pos, double* vel, const double* mass, double m_star, double dt,
               double n1, double n2, double* rcrit_row, double* out_acc, int32_t* out_pairs, int32_t* out_npairs);

#ifdef __cplusplus
}
#endif
#endif /* GENGA_STEP_H */
