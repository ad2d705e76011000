/*
 * genga_senc.h -- C ABI of the close-encounter detection after the drift and of the multi-level step
 * (the recursive function SEnc, "Symplectic Encounters") of arXiv 2201.10058, App. A (
 * SURVEY.md 8(f) NEXT-2 first half and NEXT-4).
 *
 * Works on the context of genga_kick.h (its N bodies, G, enc_factor, stream); only ENQUEUES kernels and
 * never synchronises; all pointers are DEVICE pointers, 16-byte aligned, owned by the caller.  There is no
 * CPU fallback.  Return codes and genga_kick_strerror as in genga_kick.h.
 */
#ifndef GENGA_SENC_H
#define GENGA_SENC_H

#include "genga_kick.h"

#ifdef __cplusplus
extern "C" {
#endif

/*
 * Close-encounter detection (App. A: "FG(dt); if (close-encounter candidates): close-encounter
 * detection").  PAPER.md prints no criterion; reading G16 (parity with the PAPER unpinned, parity
 * with the oracle bit-exact): a candidate {i, j} is a close-encounter pair of the step if the minimum over
 * the step of the cubic Hermite interpolant of |q_j - q_i|^2 -- through its values and time derivatives
 * 2 (q_j - q_i).(v_j - v_i) before and after the drift -- is < (enc_factor * max(rc_i, rc_j))^2.
 *
 *   pos0, vel0   [3][N] state before the drift            pos1, vel1   [3][N] state after it
 *   rcrit_row    [N] the critical radii of the level       h            the drift's time step
 *   enc_factor   scales the radius (1.0: the critical radius itself)
 *   in_pairs     [in_pair_rows][2] candidates (e.g. out_pairs of genga_kick); in_n_pairs: device pointer to
 *                ONE int32, their number (clipped to in_pair_rows)
 *   out_pairs    [pair_capacity of the context][2]: the close-encounter pairs, i < j, arbitrary order
 *   out_npairs   [N + 1]: close-encounter pairs per body, then [N] = their total (rows beyond the capacity
 *                are counted, not written)
 * The decision is taken in IEEE binary64 without contraction, in the order the oracle states it.
 * A row with an index outside [0, N) or i == j is ignored and sets GENGA_KICK_STATUS_BAD_PAIR (16).
 * Errors: E_NULL, E_ALIGN, E_SIZE (in_pair_rows < 0, enc_factor <= 0), E_CUDA.
 */
int genga_detect(genga_kick_ctx* ctx, const double* pos0, const double* vel0, const double* pos1, const double* vel1,
                 const double* rcrit_row, double enc_factor, double h, const int32_t* in_pairs,
                 const int32_t* in_n_pairs, int64_t in_pair_rows, int32_t* out_pairs, int32_t* out_npairs);

#define GENGA_KICK_STATUS_LIST_CLIPPED 128   /* genga_multilevel_step: a candidate or close-encounter list was longer than
                                               the context's pair_capacity; the rows beyond it were not seen by the
                                               levels below -- repeat the step with a larger capacity               */

typedef struct {
    int32_t slevels;    /* number of symplectic levels, 1 .. 4 (1: the original hybrid scheme; the context needs
                           max_level >= slevels - 1); genga_steps also takes 0: no encounter branch                                                              */
    int32_t substeps;   /* sub-steps per level >= 1 ("two, four, or 10, but any other number is also possible",
                           PAPER.md:619); ignored for slevels == 1                                                */
    int32_t detect;     /* 1: close-encounter detection as genga_detect (threshold: the critical radius itself);
                           0: every candidate of a pre-check counts as a close-encounter pair                     */
    int32_t reserved;
    double  n1, n2;     /* eq. 5 (3 and 0.4)                                                         */
    double  tol;        /* Bulirsch-Stoer tolerance (genga_bs.h)                                                  */
} genga_senc_config;

/*
 * One step of the multi-level scheme (App. A), on the device with no host round trip:
 *
 *     Rcrit(dt); Kick(dt/2) + pre-check; HC(dt/2); FG(dt); close-encounter detection
 *     SLevels > 1:  SEnc(dt, 1.0, 0)            else:  grouping; Bulirsch-Stoer(dt)
 *     HC(dt/2); Kick(dt/2)
 *
 *     SEnc(dt, ds, SLevel):  groupS;  SLevel += 1;  ds *= substeps
 *       for s < substeps:  RcritS;  KickS(dt/ds/2);  FGS(dt/ds);  detection;
 *                          SLevel < SLevels - 1 ?  SEnc(dt, ds, SLevel)  :  grouping; Bulirsch-Stoer(dt/ds)
 *                          KickS(dt/ds/2)
 *
 * Reading G17: level l >= 1 works on the close-encounter pairs of level l - 1 and the bodies in
 * them; these restart from their state before the upper level's drift; RcritS writes row l of eq. 5 at
 * dt / substeps^l from the current velocities; KickS is genga_kick_list at level l; the Bulirsch-Stoer phase
 * of the deepest level carries W_BS = prod_{k < SLevels} (1 - K_k).  The paper's "if (close-encounters)"
 * tests are not taken on the host: every kernel of the fixed launch sequence reads its counts on the device and
 * does nothing on an empty list (the sequence can be captured in a CUDA graph).
 *
 *   pos, vel     [3][N] advanced in place               mass [N]
 *   out_pairs / out_npairs   the candidates of the first kick, as genga_kick writes them
 *   A list longer than pair_capacity is clipped (as genga_kick does) and GENGA_KICK_STATUS_LIST_CLIPPED is set.
 *   out_stats    [slevels][4] int32 or NULL: per level, summed over its sub-steps: candidate pairs,
 *                close-encounter pairs, groups handed to Bulirsch-Stoer, bodies in them
 *   out_acc      [3][N] acceleration of the closing kick, or NULL
 * Errors: E_NULL, E_ALIGN, E_SIZE (slevels outside 1..4, substeps < 1, tol <= 0, m_star <= 0), E_LEVEL
 * (slevels - 1 > max_level of the context), E_NOMEM, E_CUDA.
 */
int genga_multilevel_step(genga_kick_ctx* ctx, double* pos, double* vel, const double* mass, double m_star, double dt,
                          const genga_senc_config* cfg, double* out_acc, int32_t* out_pairs, int32_t* out_npairs,
                          int32_t* out_stats);

#define GENGA_KICK_STATUS_RCRIT_JUMP 256   /* genga_steps: a body's critical radius grew by more than 1/64 from one step
                                             to the next, more than the merged kick's candidate list allows for:
                                             repeat from the state before the call with single steps               */

/*
 * n_steps consecutive steps of the scheme above in one call, with the closing Kick(dt/2) of every step but the last
 * and the opening Kick(dt/2) + pre-check of the next MERGED into one pass over the pairs: both act on the same
 * positions (App. A, repeated) and differ only in the critical radii -- the next step's Rcrit(dt) is
 * taken from the velocities after the closing kick -- i.e. only in the pairs inside a critical radius.  The far field
 * is summed once and the listed pairs are evaluated twice (rc of the step that ends, then rc of the step that begins,
 * with its pre-check).  The result equals n_steps calls of genga_multilevel_step (cfg->slevels >= 1; 1 = the hybrid
 * step of genga_bs.h when cfg->detect == 0) or of genga_step (cfg->slevels == 0: no encounter branch, cfg->n1 / n2
 * used, cfg->tol / substeps / detect ignored) up to the rounding of the far-field sums; a step costs one all-pairs
 * pass instead of two.
 *   out_pairs / out_npairs   the candidates of the LAST step's opening kick
 *   out_stats                [slevels][4] summed over all steps, or NULL
 *   out_acc                  acceleration of the final closing kick, or NULL
 * Errors: as genga_multilevel_step; E_SIZE also for n_steps < 1.
 */
int genga_steps(genga_kick_ctx* ctx, double* pos, double* vel, const double* mass, double m_star, double dt,
                int32_t n_steps, const genga_senc_config* cfg, double* out_acc, int32_t* out_pairs, int32_t* out_npairs,
                int32_t* out_stats);

#ifdef __cplusplus
}
#endif
#endif /* GENGA_SENC_H */
