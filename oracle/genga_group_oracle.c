/*
 * CPU ORACLE for the grouping of close-encounter pairs.
 *                                                        *** TEST INFRASTRUCTURE ONLY ***
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * call this file.  It shares no code, header, table or helper with the CUDA path.
 *
 * Definition ("sort them into independent close-encounter groups ... bodies [that]
 * have multiple close-encounter pairs ... need to be linked together in a bigger close-encounter
 * group"; "GENGA sorts all close-encounter pairs into independent groups, which can
 * be integrated in parallel"): the groups are the CONNECTED COMPONENTS of the graph whose vertices
 * are the bodies and whose edges are the pairs of the list.  A body without a pair is in no group.
 * The partition is unique; it is written in a canonical form so that it can be compared bit for bit:
 *   group_of[i] = smallest body index of i's group, -1 if i has no pair
 *   members     = the bodies that are in a group, sorted by (group_of, body index)
 *   offsets[g]  = start of group g in members, groups in ascending order of their smallest body;
 *                 offsets[n_groups] = n_members
 * Plain sequential union-find, then one pass that names every tree after its smallest vertex.
 *
 * PINS (tests/test_group_oracle_pins.py): scipy.sparse.csgraph.connected_components on seeded
 * random graphs; the Fig. 7 ring (4N pairs -> ONE group of N); disjoint pairs
 * (N/2 groups of 2); a chain; a star; the empty list; duplicate and reversed pairs.
 */
#include <stdint.h>
#include <stdlib.h>

static int32_t find_root(int32_t *parent, int32_t x)
{
    while (parent[x] != x) { parent[x] = parent[parent[x]]; x = parent[x]; }
    return x;
}

/* returns n_groups; *n_members and *max_size are filled.  members [N], offsets [N + 1]. */
int64_t genga_oracle_group(int64_t N, const int32_t *pairs, int64_t n_pairs, int32_t *group_of,
                           int32_t *members, int32_t *offsets, int64_t *n_members, int64_t *max_size)
{
    int32_t *parent = (int32_t *)malloc((size_t)(N > 0 ? N : 1) * sizeof(int32_t));
    int32_t *smallest = (int32_t *)malloc((size_t)(N > 0 ? N : 1) * sizeof(int32_t));
    char *in_pair = (char *)calloc((size_t)(N > 0 ? N : 1), 1);
    for (int64_t i = 0; i < N; i++) parent[i] = (int32_t)i;
    for (int64_t p = 0; p < n_pairs; p++) {
        const int32_t u = pairs[2 * p], v = pairs[2 * p + 1];
        in_pair[u] = in_pair[v] = 1;
        const int32_t ru = find_root(parent, u), rv = find_root(parent, v);
        if (ru != rv) parent[ru] = rv;
    }
    /* name every tree after its smallest vertex: vertices are visited in ascending order, so the
     * first visitor of a root is the smallest vertex of that tree */
    for (int64_t i = 0; i < N; i++) smallest[i] = -1;
    for (int64_t i = 0; i < N; i++) {
        const int32_t r = find_root(parent, (int32_t)i);
        if (smallest[r] < 0) smallest[r] = (int32_t)i;
        group_of[i] = in_pair[i] ? smallest[r] : -1;
    }
    /* members by (group, body): groups in ascending order of their name; a counting pass per group
     * start keeps it plain: size[name] first, then offsets, then fill in ascending body order */
    int64_t *size = (int64_t *)calloc((size_t)(N > 0 ? N : 1), sizeof(int64_t));
    int64_t *cursor = (int64_t *)malloc((size_t)(N > 0 ? N : 1) * sizeof(int64_t));
    for (int64_t i = 0; i < N; i++) if (group_of[i] >= 0) size[group_of[i]]++;
    int64_t ng = 0, nm = 0, mx = 0;
    for (int64_t g = 0; g < N; g++) {
        if (size[g] == 0) continue;
        offsets[ng++] = (int32_t)nm;
        cursor[g] = nm;
        nm += size[g];
        if (size[g] > mx) mx = size[g];
    }
    offsets[ng] = (int32_t)nm;
    for (int64_t i = 0; i < N; i++) if (group_of[i] >= 0) members[cursor[group_of[i]]++] = (int32_t)i;
    free(parent); free(smallest); free(in_pair); free(size); free(cursor);
    if (n_members) *n_members = nm;
    if (max_size) *max_size = mx;
    return ng;
}
