/*
 * genga_group.h -- C ABI of the grouping of close-encounter pairs.
 *
 * "The integrator needs to search for close-encounter pairs at each time step and to sort them
 * into independent close-encounter groups ... bodies [that] have multiple close-encounter pairs
 * ... need to be linked together in a bigger close-encounter group" (arXiv 2201.10058 sec. 2,
 * PAPER.md:78); "GENGA sorts all close-encounter pairs into independent groups, which can be
 * integrated in parallel" (sec. 6.1); App. A `grouping`.
 *
 * The groups are the connected components of the graph whose vertices are the bodies and whose
 * edges are the rows of the pair list genga_kick (or genga_step) has written.  The partition is
 * unique and is returned in a canonical form, so the result is a fixed function of the pair SET
 * (the order of the list, which is arbitrary -- PAPER.md:1047 -- does not matter; no 'Serial
 * Grouping' sort is needed):
 *
 *   group_of[i]  smallest body index of the group body i is in; -1 if i is in no pair
 *   members      the bodies that are in a group, sorted by (group, body index)
 *   offsets[g]   group g is members[offsets[g] .. offsets[g+1]); groups in ascending order of
 *                their smallest body; offsets[n_groups] = n_members
 *   summary[0..3] n_groups, n_members, size of the largest group, pair rows used
 *
 * Works on the context of genga_kick.h (its N bodies and stream); only enqueues kernels and
 * never synchronises; all pointers are DEVICE pointers owned by the caller.
 */
#ifndef GENGA_GROUP_H
#define GENGA_GROUP_H

#include "genga_kick.h"

#ifdef __cplusplus
extern "C" {
#endif

#define GENGA_KICK_STATUS_BAD_PAIR 16   /* a pair row held an index outside [0, N): row ignored */

/*
 *   pairs      [pair_rows][2] int32, as written by genga_kick (any order, duplicates allowed)
 *   n_pairs    device pointer to ONE int32: the number of pairs (e.g. out_npairs + N of genga_kick;
 *              the TRUE total there may exceed the rows written: it is clipped to pair_rows, and
 *              summary[3] tells how many rows were used)
 *   pair_rows  rows readable in `pairs`
 *   group_of   [N]       members [N]       offsets [N + 1]       summary [4]     (int32, 16-byte aligned)
 * Errors: E_NULL, E_ALIGN, E_SIZE (pair_rows < 0), E_CUDA.
 */
int genga_group(genga_kick_ctx* ctx, const int32_t* pairs, const int32_t* n_pairs, int64_t pair_rows,
                int32_t* group_of, int32_t* members, int32_t* offsets, int32_t* summary);

#ifdef __cplusplus
}
#endif
#endif /* GENGA_GROUP_H */
