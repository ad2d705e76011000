/*
 * genga_kick_static.h -- the list kick (KickS) for callers that must not allocate.
 *
 * genga_kick_init / genga_kick_list (genga_kick.h) keep their scratch in a context that cudaMalloc's it.
 * Code under CUDA stream capture, tight serving loops and harnesses that forbid cudaMalloc cannot create
 * one.  genga_kick_list_static is the same operation -- App. A, PAPER.md:1003-1021 (KickS), weights of
 * eq. 62-63, pre-check of App. A PAPER.md:989 -- with NO context: its scratch (the
 * fixed-point accumulators of the near terms and their "touched" flags) is a file-scope
 * `static __device__` array inside the library.
 *
 *   - It calls no cudaMalloc, cudaFree or allocating library routine, ever: memsets and two kernels on the
 *     caller's stream.  The first call on a device resolves the array's device address
 *     (cudaGetSymbolAddress, once per device, with that device current); make that first call outside a
 *     stream capture.
 *   - The array is GENGA_KICK_STATIC_SCRATCH_BYTES (9.25 MiB) and serves N = n_massive + n_test up to
 *     GENGA_KICK_STATIC_MAX_BODIES (65,536: BASELINE.json configs[3]).  Every GPU that loads the library
 *     holds it until the process exits.  A larger N is refused with GENGA_KICK_E_STATIC_MAX: use a context.
 *   - ALL calls on a device share the one array, and it keeps the last call's contents.  Each call clears
 *     the part it uses first, on its stream.  Calls that OVERLAP on the GPU (two streams, two host threads
 *     with their own streams, a captured graph replayed beside a direct call) RACE on it and give wrong
 *     sums without any error: serialise them (one stream, or events).  genga_kick_list on a context has its
 *     own scratch and may overlap with anything.
 *
 * The results are those of genga_kick_list bit for bit (the same kernels; the sums are fixed-point, hence
 * independent of any order): tests/test_zz_no_alloc.py.
 */
#ifndef GENGA_KICK_STATIC_H
#define GENGA_KICK_STATIC_H

#include "genga_kick.h"

#ifdef __cplusplus
extern "C" {
#endif

#define GENGA_KICK_STATIC_MAX_BODIES 65536
/* [3 components][6 limbs][MAX] 64-bit accumulators + [MAX] 32-bit flags */
#define GENGA_KICK_STATIC_SCRATCH_BYTES (GENGA_KICK_STATIC_MAX_BODIES * (3 * 6 * 8 + 4))
#define GENGA_KICK_E_STATIC_MAX (-7)   /* N exceeds GENGA_KICK_STATIC_MAX_BODIES: the static scratch cannot hold it */

/*
 * All pointers are DEVICE pointers on the current device, 16-byte aligned, owned by the caller:
 *   pos [3][N], mass [N], rcrit [changeover_level + 1][N]   inputs, as genga_kick
 *   vel [3][N] or NULL      in/out: v += dt a
 *   out_acc [3][N] or NULL  out: a (bodies in no listed pair get 0); vel and out_acc not both NULL
 *   in_pairs [in_pair_rows][2], in_n_pairs (ONE int32: listed pairs, clipped to in_pair_rows): as genga_kick_list
 *   out_pairs [pair_capacity][2] (NULL allowed iff pair_capacity == 0), out_npairs [N + 1]: as genga_kick
 *   status  ONE int32, out: cleared, then the GENGA_KICK_STATUS_* bits of this call (1 coincident bodies,
 *           4 fixed-point range, 16 bad list row); read it after the stream has drained
 *   n_massive, n_test, G, enc_factor, tp_mode (0 or 1: TP 1, 2: TP 2): what genga_kick_config holds for a context
 *   cuda_stream  a cudaStream_t (NULL: the default stream); the call returns without synchronising
 * Errors: E_NULL, E_ALIGN, E_SIZE (negative sizes, N == 0, tp_mode outside 0..2), E_LEVEL (level < 0 or > 62),
 * GENGA_KICK_E_STATIC_MAX (N > GENGA_KICK_STATIC_MAX_BODIES; nothing is launched), E_CUDA (no sm_100 device
 * current, or a CUDA call failed).
 */
int genga_kick_list_static(const double* pos, double* vel, const double* mass, const double* rcrit,
                           int64_t n_massive, int64_t n_test, int32_t changeover_level, int32_t tp_mode,
                           double G, double enc_factor, double dt,
                           const int32_t* in_pairs, const int32_t* in_n_pairs, int64_t in_pair_rows,
                           double* out_acc, int32_t* out_pairs, int64_t pair_capacity, int32_t* out_npairs,
                           int32_t* status, void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif
