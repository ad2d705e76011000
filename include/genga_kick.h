/*
 * genga_kick.h -- C ABI of the B200-native GENGA kick + close-encounter pre-check.
 *
 * The one operation behind this boundary is the interaction part H_B of the hybrid symplectic
 * integrator of arXiv 2201.10058 (eq. 3; App. A PAPER.md:986-992 "Kick(dt/2),
 * close-encounter pre-check"):
 *
 *   a_i = sum_{j in [0, n_massive), j != i}  G m_j W_L(r_ij) (x_j - x_i) / r_ij^3
 *
 *   W_0 = K(r; rc0_ij)
 *   W_L = prod_{k<L} [1 - K(r; rck_ij)] * K(r; rcL_ij)         eq. 62-63
 *   K(r; rc): y = (r - 0.1 rc)/(0.9 rc); 0 for y <= 0; 1 for y >= 1; else y^2/(2y^2 - 2y + 1)
 *   rck_ij = max(rcrit[k][i], rcrit[k][j])                     eq. 5
 *   pre-check: (i, j) is an encounter pair iff r_ij^2 < (enc_factor * rcL_ij)^2   (strict)
 *
 * Bodies [0, n_massive) interact fully; bodies [n_massive, n_massive + n_test) are semi-active
 * test particles: they feel the massive bodies and not each other (sec. 8.1).
 * With tp_mode = 2 ("TP 2") those that have mass also act on the massive bodies, in the sum above;
 * otherwise ("TP 1") they exert no force.  Readings of the paper where it is silent: DESIGN.md.
 *
 * All functions return 0 on success or a negative genga_kick_error.  Nothing throws, aborts or
 * prints.  Nothing falls back to the CPU: without a usable CUDA device genga_kick_init fails.
 */
#ifndef GENGA_KICK_H
#define GENGA_KICK_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    GENGA_KICK_OK        =  0,
    GENGA_KICK_E_NULL    = -1,   /* a required pointer is NULL                                   */
    GENGA_KICK_E_ALIGN   = -2,   /* a device pointer is not 16-byte aligned                      */
    GENGA_KICK_E_SIZE    = -3,   /* n_massive < 0, n_test < 0, N == 0 or N > 2^30, capacity < 0  */
    GENGA_KICK_E_LEVEL   = -4,   /* changeover_level outside [0, max_level]                      */
    GENGA_KICK_E_CUDA    = -5,   /* a CUDA call failed; genga_kick_last_cuda_error() has the text */
    GENGA_KICK_E_NOMEM   = -6    /* host allocation failed                                       */
} genga_kick_error;

/* bits of the device status word (genga_kick_status) */
#define GENGA_KICK_STATUS_COINCIDENT 1   /* two distinct bodies at the same position were met
                                            (outside the domain; that pair was skipped)          */
#define GENGA_KICK_STATUS_CAND_OVERFLOW 2 /* more pairs inside a critical radius than the library's
                                            candidate list holds (64 per body, at least 2^20): the
                                            excess pairs were evaluated on a slow path.  The results
                                            are COMPLETE; the bit only says why the call was slow  */
#define GENGA_KICK_STATUS_FX_RANGE 4     /* a changeover-weighted term outside [7e-43, 4.5e15]
                                            (or not finite) was met and left out of out_acc       */

typedef struct genga_kick_ctx genga_kick_ctx;   /* opaque; owned by the library */

typedef struct {
    int32_t n_massive;      /* fully interacting bodies: indices [0, n_massive)                    */
    int32_t n_test;         /* semi-active test particles: [n_massive, n_massive + n_test)         */
    int32_t max_level;      /* largest changeover_level that will be passed (0 = original K only)  */
    int32_t device;         /* CUDA device ordinal                                                 */
    int64_t pair_capacity;  /* rows available in out_pairs                                         */
    double  G;              /* gravitational constant; k^2, k = 0.01720209895 in AU / day / Msun   */
    double  enc_factor;     /* f in r_ij < f * rcL_ij; 1.0                                         */
    int32_t order_mode;     /* GENGA_KICK_ORDER_*: the library's INTERNAL body order (never visible
                               in the outputs; changes speed and summation order, not the contract) */
    int32_t tp_mode;        /* force terms of the semi-active particles (Fig. 14):
                               0 or 1 = "TP 1": they feel the massive bodies and exert no force;
                               2      = "TP 2": those with mass also act on the massive bodies       */
} genga_kick_config;

#define GENGA_KICK_ORDER_AUTO    0   /* spatially sorted copy when N >= 4096, caller's order below  */
#define GENGA_KICK_ORDER_CALLER  1   /* always the caller's order                                   */
#define GENGA_KICK_ORDER_SORTED  2   /* always the spatially sorted copy                            */

/*
 * How one call is cut into CTAs (host logic, no CUDA call; exported so it can be tested on a
 * machine without a GPU).  The kick is a grid of tiles (i-block x j-tile), i-major; CTA c owns
 * the contiguous tile range [c*T/n_ctas, (c+1)*T/n_ctas) and writes one partial-sum segment per
 * i-block it touches; a second pass adds the segments of each i-block in ascending CTA order
 * (fixed order => bit-reproducible).
 */
typedef struct {
    int32_t threads;        /* threads per CTA                                                     */
    int32_t i_per_thread;   /* i-bodies owned by one thread                                        */
    int32_t i_block;        /* = threads * i_per_thread                                            */
    int32_t j_tile;         /* j-bodies per shared-memory tile                                     */
    int32_t m_pad;          /* records [0, m_pad): massive bodies + padding; test particles follow  */
    int32_t n_i_blocks;     /* ceil(n_i / i_block), n_i = n_test ? m_pad + n_test : n_massive      */
    int32_t n_j_tiles;      /* ceil(n_massive / j_tile)                                            */
    int64_t n_tiles;        /* T = n_i_blocks * n_j_tiles                                          */
    int32_t n_ctas;         /* CTAs launched (a multiple of the SM count unless T is smaller; up to
                               four waves of resident CTAs when every CTA keeps >= 16 tiles)      */
    int32_t max_segs;       /* most i-blocks any CTA touches                                       */
    int64_t n_rec;          /* records allocated (n_i rounded up to a multiple of 1024)            */
    int64_t partial_doubles;/* doubles of scratch for the partial sums                             */
    /* symmetric plans only (genga_kick_make_plan_sym; 0 otherwise) */
    int32_t symmetric;      /* 1: massive x massive with every unordered pair evaluated once: row I (i-block I)
                               holds only the j-tiles jt >= I * tiles_per_iblock; tiles numbered row-major  */
    int32_t tiles_per_iblock;/* i_block / j_tile: the first that many tiles of a row overlap the i-block
                               (diagonal tiles, one-sided); the rest give force and reaction           */
    int64_t react_doubles;  /* doubles of scratch for the reaction partial sums: n_tiles * 3 * j_tile */
} genga_kick_plan;

/* Fill *plan for a problem of n_massive + n_test bodies at changeover level `level` on a device
 * with num_sms multiprocessors.  Errors: E_NULL, E_SIZE, E_LEVEL (level < 0). */
int genga_kick_make_plan(int32_t n_massive, int32_t n_test, int32_t level, int32_t num_sms,
                         genga_kick_plan* plan);
/* TP 2 only: the plan of the second pass of a level-0 kick, massive bodies (i) x semi-active
 * particles (j), same tile / CTA / partial-sum scheme.  Errors: E_NULL, E_SIZE. */
int genga_kick_make_plan_tp2(int32_t n_massive, int32_t n_test, int32_t num_sms, genga_kick_plan* plan);
/* Level 0, massive x massive, Newton's third law: each unordered pair is evaluated once (eq. 3 is symmetric in i, j:
 * PAPER.md:63-64), the j-side sums are written per tile and added in ascending row order by the reduction pass.
 * plan->n_ctas == 0 if the library does not use it for this size (n_massive below 24,576, or the reaction scratch
 * above 2 GiB).  Test particles are not part of it (they take the one-sided rows of genga_kick_make_plan_tprows).
 * Errors: E_NULL, E_SIZE. */
int genga_kick_make_plan_sym(int32_t n_massive, int32_t n_test, int32_t num_sms, genga_kick_plan* plan);
/* The one-sided rows of the semi-active particles (i = particles, j = massive bodies) when the massive bodies take the
 * symmetric plan: same tile / CTA / partial-sum scheme as genga_kick_make_plan, i-blocks counted from record m_pad.
 * Errors: E_NULL, E_SIZE. */
int genga_kick_make_plan_tprows(int32_t n_massive, int32_t n_test, int32_t num_sms, genga_kick_plan* plan);
/* Symmetric plans: the first tile of every CTA, cta_first_tile[0 .. n_ctas] (the last entry is n_tiles).  The ranges
 * are contiguous and ascending but not equally long: they balance a cost model in which a diagonal tile (ordered
 * pairs, mostly inside filter radii) weighs 1.4 symmetric tiles.  Errors: E_NULL, E_SIZE (not a symmetric plan in use). */
int genga_kick_plan_sym_table(const genga_kick_plan* plan, int64_t* cta_first_tile);
/* Symmetric plans: first tile of row `row` (row = n_i_blocks gives n_tiles) and the row of tile t. */
int64_t genga_kick_plan_sym_row_begin(const genga_kick_plan* plan, int32_t row);
int32_t genga_kick_plan_sym_row_of(const genga_kick_plan* plan, int64_t t);
/* Tile range [*t0, *t1) of CTA `cta` under *plan.  Errors: E_NULL, E_SIZE. */
int genga_kick_plan_cta_range(const genga_kick_plan* plan, int32_t cta, int64_t* t0, int64_t* t1);
/* First and last CTA whose range meets i-block `ib`.  Errors: E_NULL, E_SIZE. */
int genga_kick_plan_iblock_ctas(const genga_kick_plan* plan, int32_t ib, int32_t* c_first, int32_t* c_last);

/* Create a context on cfg->device: allocates the library's scratch (packed j-bodies, partial
 * sums, host-call staging is allocated lazily).  *out_ctx is written only on success.
 * Errors: E_NULL, E_SIZE, E_LEVEL, E_CUDA (no device, wrong device, out of memory). */
int genga_kick_init(const genga_kick_config* cfg, genga_kick_ctx** out_ctx);

/* Stream the following genga_kick calls enqueue on (a cudaStream_t, e.g.
 * torch.cuda.current_stream().cuda_stream; NULL = the default stream).  Not owned. */
int genga_kick_set_stream(genga_kick_ctx* ctx, void* cuda_stream);

/*
 * One kick + pre-check.  N = n_massive + n_test.  Every array is DEVICE memory owned by the
 * caller, 16-byte aligned, and must stay valid until the stream has run the call.  The call only
 * enqueues kernels on the context's stream; it never synchronises.
 *
 *   pos        [3][N] SoA (x[0..N), y[0..N), z[0..N)), heliocentric positions        (read)
 *   vel        [3][N] SoA or NULL; if non-NULL, v += dt * a in place (what Kick(dt/2) of
 *              App. A does with dt = half the step)                                   (read/write)
 *   mass       [N]                                                                    (read)
 *   rcrit      [changeover_level + 1][N]: row k = r_crit,i at time step dt / s^k      (read)
 *   out_acc    [3][N] SoA accelerations; NULL allowed only if vel is non-NULL         (write)
 *   out_pairs  [pair_capacity][2] int32, each unordered encounter pair once as (lo, hi),
 *              rows in arbitrary order; may be NULL if pair_capacity == 0 (write)
 *   out_npairs [N + 1] int32: [i] = number of encounter partners of body i (a massive body also
 *              counts its test-particle partners); [N] = TRUE number of pairs found.  If
 *              [N] > pair_capacity the rows beyond capacity were dropped (never written out of
 *              bounds) and the caller re-calls with a larger buffer.                  (write)
 *
 * out_acc and out_npairs are bit-reproducible from call to call; out_pairs is a set.
 * Errors: E_NULL, E_ALIGN, E_LEVEL, E_CUDA.
 */
int genga_kick(genga_kick_ctx* ctx,
               const double* pos, double* vel, const double* mass, const double* rcrit,
               int32_t changeover_level, double dt,
               double* out_acc, int32_t* out_pairs, int32_t* out_npairs);

/*
 * What a call may keep from the calls before it (the kicks of several changeover levels of one step act on the same
 * positions; sec. 7.1, eq. 62-63):
 *   on = GENGA_KICK_REUSE_OFF   (default) every call sorts and searches: its outputs are a fixed function of its inputs alone.
 *   on = GENGA_KICK_REUSE_ORDER genga_kick keeps the internal body order of the last call that sorted instead of sorting
 *        again: for consecutive calls on unchanged or little-changed positions.  The internal order is never visible
 *        and never changes a result beyond the order of its sums; it only decides how many tiles the culling can clear.
 *   on = GENGA_KICK_REUSE_LIST  as GENGA_KICK_REUSE_ORDER, and the caller states that `pos` of every level >= 1 call made
 *        under this setting is BIT-IDENTICAL to `pos` of the last level-0 call on this context: such a kick also skips
 *        its neighbour search and evaluates the list of near pairs the level-0 kick has left (the pairs inside
 *        max(rc0, f rc0) of either body: a superset of the pairs inside max(rc0, f rcL), outside of which W_L = 0 and
 *        there is no encounter, as long as no body's filter radius at level L exceeds its level-0 one -- checked per
 *        body on the device; if one does, or if no level-0 list is at hand, that kick searches all pairs itself).
 *        Results are those of GENGA_KICK_REUSE_ORDER bit for bit (the near terms are summed exactly; the order of the
 *        rows of out_pairs is arbitrary in every mode).  Changed positions under this setting give wrong results
 *        without a status bit: the library cannot see it.
 * Errors: E_NULL, E_SIZE (on outside 0..2).
 */
#define GENGA_KICK_REUSE_OFF 0
#define GENGA_KICK_REUSE_ORDER 1
#define GENGA_KICK_REUSE_LIST 2
int genga_kick_set_order_reuse(genga_kick_ctx* ctx, int32_t on);

/*
 * The same call with HOST arrays (same shapes; any alignment; vel and out_acc may be NULL as
 * above, out_pairs may be NULL): copies the inputs to library-owned device buffers, runs
 * genga_kick, copies the results back and synchronises the stream before returning.  At most
 * min([N], pair_capacity) pair rows are copied back.  Errors: as genga_kick.
 */
int genga_kick_host(genga_kick_ctx* ctx,
                    const double* pos, double* vel, const double* mass, const double* rcrit,
                    int32_t changeover_level, double dt,
                    double* out_acc, int32_t* out_pairs, int32_t* out_npairs);

/*
 * KickS (App. A: "KickS ... similar to the original functions, but applied only to
 * the relevant bodies in each symplectic level"; groupS "extracts all relevant close-encounter pairs
 * from the upper symplectic level"): the kick of level `changeover_level` over the pairs of a LIST
 * instead of over all pairs, plus the level pre-check of the listed pairs:
 *     a_i = sum over listed pairs {i, j} of  G m_j W_L(r_ij) (x_j - x_i) / r_ij^3      (both members of a pair)
 *     out_pairs / out_npairs: the listed pairs with r_ij^2 < (f rcL_ij)^2, as genga_kick writes them
 * Since W_L = 0 for r >= rc0_ij (L >= 1), this equals genga_kick at level L whenever the list holds
 * every pair with r < rc0_ij -- e.g. the list genga_kick wrote at level 0 with enc_factor >= 1 for the
 * same positions -- at a cost proportional to the list instead of N^2.
 *   in_pairs    [in_pair_rows][2] int32 device, each unordered pair once (the caller's indices)
 *   in_n_pairs  device pointer to ONE int32: number of listed pairs (clipped to in_pair_rows), e.g.
 *               out_npairs + N of the call that wrote in_pairs
 *   out_pairs, out_npairs: distinct from in_pairs / in_n_pairs.  Other arguments as genga_kick.
 * Bodies in no listed pair get a = 0.  Semi-active particles: as genga_kick (tp_mode).
 * A row with an index outside [0, N) or i == j is ignored and sets GENGA_KICK_STATUS_BAD_PAIR (16).
 * Errors: E_NULL, E_ALIGN, E_SIZE (in_pair_rows < 0), E_LEVEL, E_CUDA.
 */
int genga_kick_list(genga_kick_ctx* ctx, const double* pos, double* vel, const double* mass, const double* rcrit,
                    int32_t changeover_level, double dt, const int32_t* in_pairs, const int32_t* in_n_pairs,
                    int64_t in_pair_rows, double* out_acc, int32_t* out_pairs, int32_t* out_npairs);

/* Plan the context uses at `changeover_level` (what genga_kick will launch). */
int genga_kick_get_plan(const genga_kick_ctx* ctx, int32_t changeover_level, genga_kick_plan* plan);

/* Synchronise the stream and read the device status word (GENGA_KICK_STATUS_* bits, OR-ed over
 * all calls since init) into *status. */
int genga_kick_status(genga_kick_ctx* ctx, int32_t* status);

/* Kernel launches enqueued by the context since init (for the bench's launch count). */
int64_t genga_kick_launch_count(const genga_kick_ctx* ctx);

/* Measurement aid: with on != 0 every following genga_kick records a CUDA event pair around its
 * pair-loop kernel (the N^2 part, rows a1-a6 of SURVEY.md 8(a)) on the context's stream.
 * genga_kick_last_pair_loop_ms waits for the pair of the most recent call at `changeover_level`
 * and returns that kernel's duration in *ms (it synchronises on the event, like
 * genga_kick_status / genga_kick_host synchronise on the stream).
 * Errors: E_NULL, E_LEVEL, E_NOMEM, E_CUDA; E_SIZE if timing is off or no such call was made. */
int genga_kick_enable_timing(genga_kick_ctx* ctx, int32_t on);
int genga_kick_last_pair_loop_ms(genga_kick_ctx* ctx, int32_t changeover_level, float* ms);

/* Free the context and its scratch.  NULL is allowed. */
int genga_kick_free(genga_kick_ctx* ctx);

/* Static text for an error code. */
const char* genga_kick_strerror(int code);
/* Text of the last CUDA error seen by this context ("" if none); valid until the next call. */
const char* genga_kick_last_cuda_error(const genga_kick_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* GENGA_KICK_H */
