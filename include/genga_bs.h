/*
 * genga_bs.h -- C ABI of the Bulirsch-Stoer integration of close-encounter groups.
 *
 * "We also use a Bulirsch-Stoer ... method to resolve the close-encounter part" (arXiv 2201.10058 sec. 2,
 * PAPER.md:47); "All particles in a given close-encounter group need to be integrated synchronously"
 * (sec. 6.1); App. A `Bulirsch-Stoer(dt)`.  For every group of genga_group the
 * part H_A of the Hamiltonian (eq. 2) restricted to the group's bodies is integrated over
 * dt, starting from the state BEFORE the Kepler drift FG:
 *
 *     dq_i/dt = v_i
 *     dv_i/dt = - G m_star q_i / |q_i|^3 + sum_{j in group, j != i} G m_j W_BS(r_ij) (q_j - q_i) / r_ij^3
 *     W_BS    = prod_{k < nlevels} [1 - K(r_ij; max(rcrit[k][i], rcrit[k][j]))]          (eq. 62-63)
 *
 * (nlevels = 1: the complement of the kick's weight).  The result REPLACES the Kepler-drifted state of
 * the group's bodies; bodies in no group are not touched.
 *
 * Method (the paper names it and refers to Grimm & Stadel 2014; reading G15): Gragg-Bulirsch-
 * Stoer -- modified midpoint with 2, 4, .., 16 sub-steps, polynomial extrapolation in h^2, relative error
 * per body in position and velocity <= tol, one step size for the whole group (halved on failure, doubled
 * after fast convergence).  Groups of up to 8 bodies: one warp per group, one lane per body, eight groups per thread
 * block, the force sum in member order; 9 .. 32 bodies: one thread block per group, eight lanes per body (together
 * BS-B of Table 2); 33 .. 256 bodies: one thread-block cluster (8 x 256 threads) per group, eight
 * lanes per body, positions exchanged through distributed shared memory (BS-A); many groups side by side.  From 9
 * bodies on the force sum of a body is taken in eight interleaved partial sums combined in a fixed tree (the oracle
 * states the order).  Larger groups: cooperative launches of co-resident thread blocks of 256 threads, eight lanes per
 * body, positions exchanged through L2 with one barrier per force evaluation (the paper's BS-M regime, PAPER.md:595-597,
 * with the sub-steps kept on the device instead of controlled from the host): groups of up to 512 and of up to 2048
 * bodies several at a time (the grid cut into teams of 16 / 64 blocks, a team per group with a barrier of its own),
 * larger ones one after the other over the whole grid -- with 8, 4, 2 or 1 lanes per body as the grid holds them (9472 /
 * 18,944 / 37,888 / 75,776 bodies on 148 SMs); beyond that GENGA_KICK_STATUS_GROUP_TOO_LARGE is set and the group keeps
 * the state already in pos / vel.  In these regimes a body only evaluates the partners on its NEIGHBOUR LIST (built at
 * the start of the group from the straight-line relative motion over dt; a pair outside the lists stays outside every
 * critical radius and contributes exactly 0, as in the all-pairs sum: n x a few terms instead of n^2 per force
 * evaluation).  The lists of a block's bodies are pooled and walked by all its warps, 32 entries at a time; a listed
 * pair's factor prod_k (1 - K_k) / r^3 is evaluated as one quotient, prod (1 - y_k)^2 / (r^3 prod (2 y_k^2 - 2 y_k + 1)),
 * from reciprocal seeds refined to < 2^-58 (the same function of r and the radii as the literal form, a few units in the
 * last place apart; the order of a body's sum is a fixed function of its list).  Groups whose lists do not fit the
 * scratch take the all-pairs sum with the literal form.  A pair with r^2 >= rc0^2 (1 + 2^-20) is dismissed after 8 FP64
 * instructions in every regime.
 *
 * Works on the context of genga_kick.h (its N, G, stream); only enqueues; all pointers are DEVICE pointers.
 */
#ifndef GENGA_BS_H
#define GENGA_BS_H

#include "genga_kick.h"

#ifdef __cplusplus
extern "C" {
#endif

#define GENGA_KICK_STATUS_GROUP_TOO_LARGE 32   /* a group larger than the co-resident grid was left as it was */
#define GENGA_KICK_STATUS_BS_NOT_CONVERGED 64  /* a step did not reach tol after 60 halvings: that group
                                                  stopped at its last accepted time                        */
#define GENGA_KICK_STATUS_BS_LIST_ESCAPE 512   /* a body of a group above 256 bodies strayed further than
                                                  G m_star dt^2 / |q|^2 from the straight line through its initial
                                                  state: a pair outside that group's neighbour lists may have been
                                                  missed (twice what the Sun's pull allows: never seen on a disk)    */

/*
 *   pos_in, vel_in  [3][N] state before FG (read only)          mass [N]
 *   rcrit           [nlevels][N], 1 <= nlevels <= 4
 *   members, offsets, summary   as written by genga_group (summary[0] = number of groups and summary[2] = size of the
 *                   largest group are read on the device; groups above 256 bodies are only looked for if summary[2] says so)
 *   pos, vel        [3][N] updated for the bodies of the integrated groups (may NOT alias pos_in / vel_in)
 * Errors: E_NULL, E_ALIGN, E_SIZE (nlevels outside 1..4, m_star <= 0, tol <= 0), E_CUDA.
 */
int genga_bs(genga_kick_ctx* ctx, const double* pos_in, const double* vel_in, const double* mass, const double* rcrit,
             int32_t nlevels, double m_star, double dt, double tol, const int32_t* members, const int32_t* offsets,
             const int32_t* summary, double* pos, double* vel);

/*
 * Diagnostics of the step-size control (what makes a comparison with another implementation of the same scheme
 * meaningful: two runs that took the same decisions differ by rounding only; where a decision differs -- an error
 * estimate within rounding of tol -- both results still satisfy the tolerance, and the difference is of that order).
 *   genga_bs_set_stats: every following genga_bs writes, for group g < rows (g as in `offsets`), the int32 row
 *       (accepted macro steps, rejected attempts = halvings, force evaluations, bodies) to group_stats[g];
 *       device memory owned by the caller, 16-byte aligned; NULL switches it off.  Groups not integrated are not written.
 *   genga_bs_totals: the same three counts and the number of groups integrated, summed over all groups and all
 *       genga_bs calls of the context (the ones inside genga_hybrid_step / genga_multilevel_step included) since
 *       init or the last reset; synchronises the stream.
 * Errors: E_NULL, E_ALIGN, E_SIZE, E_CUDA.
 */
int genga_bs_set_stats(genga_kick_ctx* ctx, int32_t* group_stats, int64_t rows);
int genga_bs_totals(genga_kick_ctx* ctx, int64_t totals[4], int32_t reset);

/*
 * The complete step of App. A on the device, no host round trip:
 *     Rcrit(dt); Kick(dt/2) + pre-check; HC(dt/2); FG(dt); grouping; Bulirsch-Stoer(dt) on the groups, from the
 *     state before FG; HC(dt/2); Kick(dt/2).
 * Every candidate pair of the pre-check is treated as an encounter pair (the paper's separate "close-encounter
 * detection" has no printed criterion; a pair that never enters its critical radius has W_BS = 0, so integrating
 * it is only extra work).  pos, vel are advanced in place; out_pairs / out_npairs: the candidates of the first
 * kick; group_of / members / offsets / summary: their groups, as genga_group writes them (all four required);
 * out_acc: acceleration of the closing kick, or NULL.  Groups too large for genga_bs keep their Kepler-drifted
 * state and set GENGA_KICK_STATUS_GROUP_TOO_LARGE.
 * Errors: E_NULL, E_ALIGN, E_SIZE, E_CUDA.
 */
int genga_hybrid_step(genga_kick_ctx* ctx, double* pos, double* vel, const double* mass, double m_star, double dt,
                      double n1, double n2, double tol, double* out_acc, int32_t* out_pairs, int32_t* out_npairs,
                      int32_t* group_of, int32_t* members, int32_t* offsets, int32_t* summary);

#ifdef __cplusplus
}
#endif
#endif /* GENGA_BS_H */
