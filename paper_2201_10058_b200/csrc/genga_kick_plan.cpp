// Host-side work decomposition of one kick (no CUDA here; see include/genga_kick.h).
//
// The pair matrix is cut into tiles: i-blocks of `i_block` bodies (all N bodies: massive first,
// then the semi-active test particles, sec. 8.1) times j-tiles of `j_tile`
// massive bodies.  Tiles are numbered i-major, t = ib * n_j_tiles + jt, and CTA c owns
// [floor(c T / C), floor((c+1) T / C)).  This splits the j-range across CTAs when N is too small
// to fill the SMs with whole i-blocks and balances to within one tile for any N.  Each CTA writes
// one partial-sum segment per i-block it touches; the reduction pass adds the segments of an
// i-block in ascending CTA order, a fixed order ("parallel reductions have a well
// defined order").
#include "../../include/genga_kick.h"
#include "genga_kick_variants.h"

#include <vector>

static int64_t cta_t0(const genga_kick_plan* p, int64_t c)
{
    return plan_tile_begin(c, p->n_tiles, p->n_ctas);
}

// Tile decomposition of an (n_i records) x (n_j records) pair matrix: picks the variant, fills the
// tile, CTA and partial-sum fields of *p (m_pad and n_rec are the caller's business).
static void fill_tiles(genga_kick_plan* p, int64_t n_i, int64_t n_j, int32_t num_sms)
{
    p->symmetric = 0; p->tiles_per_iblock = 0; p->react_doubles = 0;
    const genga_variant* vars = GENGA_VARIANTS;
    for (int v = 0; v < GENGA_N_VARIANTS; v++) {
        p->threads = vars[v].threads;
        p->i_per_thread = vars[v].i_per_thread;
        p->i_block = p->threads * p->i_per_thread;
        p->j_tile = vars[v].j_tile;
        p->n_i_blocks = (int32_t)((n_i + p->i_block - 1) / p->i_block);
        p->n_j_tiles = (int32_t)((n_j + p->j_tile - 1) / p->j_tile);
        p->n_tiles = (int64_t)p->n_i_blocks * p->n_j_tiles;
        p->n_ctas = num_sms * vars[v].ctas_per_sm;
        if (p->n_tiles >= (int64_t)GENGA_MIN_TILES_PER_CTA * p->n_ctas) {
            // Several waves of CTAs when there is enough work: the ranges stay static (every output bit is a fixed
            // function of the inputs), but the hardware hands the next range to whichever SM is free first, which
            // takes up the differences between SMs at the end of the launch (measured at N = 65,536: pair loop
            // 4.41 ms with one wave, 4.33 ms with three or more).
            int64_t waves = p->n_tiles / ((int64_t)GENGA_TILES_PER_CTA_FOR_WAVES * p->n_ctas);
            if (waves > GENGA_MAX_WAVES) waves = GENGA_MAX_WAVES;
            if (waves > 1) p->n_ctas *= (int32_t)waves;
            break;
        }
    }
    if (p->n_tiles < p->n_ctas) p->n_ctas = (int32_t)p->n_tiles;      // 0 CTAs when there is nothing to do

    // most i-blocks any CTA touches
    int32_t max_segs = 1;
    if (p->n_j_tiles > 0) {
        for (int64_t c = 0; c < p->n_ctas; c++) {
            const int64_t t0 = cta_t0(p, c), t1 = cta_t0(p, c + 1);
            if (t1 <= t0) continue;
            const int32_t segs = (int32_t)((t1 - 1) / p->n_j_tiles - t0 / p->n_j_tiles + 1);
            if (segs > max_segs) max_segs = segs;
        }
    }
    p->max_segs = max_segs;
    p->partial_doubles = (int64_t)p->n_ctas * p->max_segs * 3 * p->i_block;
}

static int plan_records(int32_t n_massive, int32_t n_test, int32_t num_sms, genga_kick_plan* p, int64_t* n_i)
{
    const int64_t N = (int64_t)n_massive + (int64_t)n_test;
    if (n_massive < 0 || n_test < 0 || N <= 0 || N > GENGA_MAX_BODIES || num_sms <= 0) return GENGA_KICK_E_SIZE;
    // records: massive bodies padded to a multiple of GENGA_M_ALIGN, then the test particles
    p->m_pad = (int32_t)(((int64_t)n_massive + GENGA_M_ALIGN - 1) / GENGA_M_ALIGN * GENGA_M_ALIGN);
    *n_i = n_test > 0 ? (int64_t)p->m_pad + n_test : (int64_t)n_massive;
    p->n_rec = (*n_i + GENGA_REC_ALIGN - 1) / GENGA_REC_ALIGN * GENGA_REC_ALIGN;
    if (p->n_rec < p->m_pad) p->n_rec = (p->m_pad + GENGA_REC_ALIGN - 1) / GENGA_REC_ALIGN * GENGA_REC_ALIGN;
    return GENGA_KICK_OK;
}

extern "C" int genga_kick_make_plan(int32_t n_massive, int32_t n_test, int32_t level, int32_t num_sms,
                                    genga_kick_plan* plan)
{
    if (!plan) return GENGA_KICK_E_NULL;
    if (level < 0) return GENGA_KICK_E_LEVEL;
    genga_kick_plan p;
    int64_t n_i = 0;
    const int rc = plan_records(n_massive, n_test, num_sms, &p, &n_i);
    if (rc != GENGA_KICK_OK) return rc;
    fill_tiles(&p, n_i, n_massive, num_sms);         // level >= 1 only uses m_pad and n_rec of the plan
    *plan = p;
    return GENGA_KICK_OK;
}

// TP 2: the second, transposed pass of the level-0 kick -- i over the massive
// records [0, n_massive), j over the test-particle records [m_pad, m_pad + n_test).
extern "C" int genga_kick_make_plan_tp2(int32_t n_massive, int32_t n_test, int32_t num_sms, genga_kick_plan* plan)
{
    if (!plan) return GENGA_KICK_E_NULL;
    genga_kick_plan p;
    int64_t n_i = 0;
    const int rc = plan_records(n_massive, n_test, num_sms, &p, &n_i);
    if (rc != GENGA_KICK_OK) return rc;
    fill_tiles(&p, n_massive, n_test, num_sms);
    *plan = p;
    return GENGA_KICK_OK;
}

extern "C" int genga_kick_make_plan_tprows(int32_t n_massive, int32_t n_test, int32_t num_sms, genga_kick_plan* plan)
{
    if (!plan) return GENGA_KICK_E_NULL;
    genga_kick_plan p;
    int64_t n_i = 0;
    const int rc = plan_records(n_massive, n_test, num_sms, &p, &n_i);
    if (rc != GENGA_KICK_OK) return rc;
    fill_tiles(&p, n_test, n_massive, num_sms);
    *plan = p;
    return GENGA_KICK_OK;
}

// Symmetric plans: first tile of every CTA under the cost model of genga_kick_variants.h; out[n_ctas] = n_tiles.
// Tile t (row-major) belongs to CTA floor(W(t) C / W_total), W(t) = cost of the tiles before t: ranges are contiguous,
// ascending and a fixed function of the plan.
static void sym_cta_table(const genga_kick_plan* p, int64_t* out)
{
    const int64_t C = p->n_ctas;
    int64_t Wtot = 0;
    for (int64_t I = 0; I < p->n_i_blocks; I++) {
        const int64_t count = p->n_j_tiles - I * p->tiles_per_iblock;
        const int64_t nd = count < p->tiles_per_iblock ? count : p->tiles_per_iblock;
        Wtot += nd * GENGA_SYM_COST_DIAG + (count - nd) * GENGA_SYM_COST_SYM;
    }
    int64_t t = 0, W = 0, next = 0;                       // next: the CTA whose first tile is looked for
    for (int64_t I = 0; I < p->n_i_blocks; I++) {
        const int64_t count = p->n_j_tiles - I * p->tiles_per_iblock;
        for (int64_t q = 0; q < count; q++, t++) {
            const int64_t owner = W * C / Wtot;
            while (next <= owner && next < C) out[next++] = t;
            W += q < p->tiles_per_iblock ? GENGA_SYM_COST_DIAG : GENGA_SYM_COST_SYM;
        }
    }
    while (next <= C) out[next++] = t;
}

extern "C" int genga_kick_plan_sym_table(const genga_kick_plan* plan, int64_t* cta_first_tile)
{
    if (!plan || !cta_first_tile) return GENGA_KICK_E_NULL;
    if (!plan->symmetric || plan->n_ctas <= 0) return GENGA_KICK_E_SIZE;
    sym_cta_table(plan, cta_first_tile);
    return GENGA_KICK_OK;
}

extern "C" int genga_kick_make_plan_sym(int32_t n_massive, int32_t n_test, int32_t num_sms, genga_kick_plan* plan)
{
    if (!plan) return GENGA_KICK_E_NULL;
    genga_kick_plan p;
    int64_t n_i = 0;
    const int rc = plan_records(n_massive, n_test, num_sms, &p, &n_i);
    if (rc != GENGA_KICK_OK) return rc;
    p.threads = GENGA_SYM_THREADS; p.i_per_thread = GENGA_SYM_IPT; p.i_block = GENGA_SYM_IBLOCK; p.j_tile = GENGA_SYM_JT;
    p.symmetric = 1;
    p.tiles_per_iblock = p.i_block / p.j_tile;
    p.n_i_blocks = (int32_t)(((int64_t)n_massive + p.i_block - 1) / p.i_block);
    p.n_j_tiles = (int32_t)(((int64_t)n_massive + p.j_tile - 1) / p.j_tile);
    p.n_tiles = sym_row_begin(p.n_i_blocks, p.n_j_tiles, p.tiles_per_iblock);
    p.react_doubles = p.n_tiles * 3 * p.j_tile;
    p.n_ctas = num_sms;                                                // one CTA of 256 threads x 8 i-bodies per SM
    const bool use = n_massive >= GENGA_SYM_MIN_BODIES && p.react_doubles * (int64_t)sizeof(double) <= GENGA_SYM_MAX_REACT_BYTES;
    if (!use) p.n_ctas = 0;
    if (p.n_tiles < p.n_ctas) p.n_ctas = (int32_t)p.n_tiles;
    int32_t max_segs = 1;
    std::vector<int64_t> tab((size_t)p.n_ctas + 1, 0);
    if (p.n_ctas > 0) sym_cta_table(&p, tab.data());
    for (int64_t c = 0; c < p.n_ctas; c++) {
        const int64_t t0 = tab[(size_t)c], t1 = tab[(size_t)c + 1];
        if (t1 <= t0) continue;
        const int32_t segs = sym_row_of(t1 - 1, p.n_j_tiles, p.tiles_per_iblock, p.n_i_blocks) -
                             sym_row_of(t0, p.n_j_tiles, p.tiles_per_iblock, p.n_i_blocks) + 1;
        if (segs > max_segs) max_segs = segs;
    }
    p.max_segs = max_segs;
    p.partial_doubles = (int64_t)p.n_ctas * p.max_segs * 3 * p.i_block;
    *plan = p;
    return GENGA_KICK_OK;
}

extern "C" int64_t genga_kick_plan_sym_row_begin(const genga_kick_plan* plan, int32_t row)
{
    if (!plan || !plan->symmetric || row < 0 || row > plan->n_i_blocks) return -1;
    return sym_row_begin(row, plan->n_j_tiles, plan->tiles_per_iblock);
}

extern "C" int32_t genga_kick_plan_sym_row_of(const genga_kick_plan* plan, int64_t t)
{
    if (!plan || !plan->symmetric || t < 0 || t >= plan->n_tiles) return -1;
    return sym_row_of(t, plan->n_j_tiles, plan->tiles_per_iblock, plan->n_i_blocks);
}

extern "C" int genga_kick_plan_cta_range(const genga_kick_plan* plan, int32_t cta, int64_t* t0, int64_t* t1)
{
    if (!plan || !t0 || !t1) return GENGA_KICK_E_NULL;
    if (cta < 0 || cta >= plan->n_ctas) return GENGA_KICK_E_SIZE;
    if (plan->symmetric) {
        std::vector<int64_t> tab((size_t)plan->n_ctas + 1, 0);
        sym_cta_table(plan, tab.data());
        *t0 = tab[(size_t)cta];
        *t1 = tab[(size_t)cta + 1];
        return GENGA_KICK_OK;
    }
    *t0 = cta_t0(plan, cta);
    *t1 = cta_t0(plan, (int64_t)cta + 1);
    return GENGA_KICK_OK;
}

extern "C" int genga_kick_plan_iblock_ctas(const genga_kick_plan* plan, int32_t ib, int32_t* c_first, int32_t* c_last)
{
    if (!plan || !c_first || !c_last) return GENGA_KICK_E_NULL;
    if (ib < 0 || ib >= plan->n_i_blocks || plan->n_j_tiles <= 0) return GENGA_KICK_E_SIZE;
    // the CTA that owns tile t is the largest c with floor(c T / C) <= t,
    // i.e. c = floor(((t + 1) C - 1) / T)
    const int64_t T = plan->n_tiles, C = plan->n_ctas;
    if (C <= 0) return GENGA_KICK_E_SIZE;
    if (plan->symmetric) {
        std::vector<int64_t> tab((size_t)C + 1, 0);
        sym_cta_table(plan, tab.data());
        const int64_t a = sym_row_begin(ib, plan->n_j_tiles, plan->tiles_per_iblock);
        const int64_t b = sym_row_begin(ib + 1, plan->n_j_tiles, plan->tiles_per_iblock) - 1;
        int32_t first = -1, last = -1;
        for (int64_t c = 0; c < C; c++) {
            if (tab[(size_t)c + 1] <= tab[(size_t)c]) continue;
            if (first < 0 && tab[(size_t)c + 1] > a) first = (int32_t)c;
            if (tab[(size_t)c] <= b) last = (int32_t)c;
        }
        *c_first = first;
        *c_last = last;
        return GENGA_KICK_OK;
    }
    const int64_t ta = plan->symmetric ? sym_row_begin(ib, plan->n_j_tiles, plan->tiles_per_iblock) : (int64_t)ib * plan->n_j_tiles;
    const int64_t tb = plan->symmetric ? sym_row_begin(ib + 1, plan->n_j_tiles, plan->tiles_per_iblock) - 1 : ta + plan->n_j_tiles - 1;
    *c_first = plan_tile_owner(ta, T, C);
    *c_last = plan_tile_owner(tb, T, C);
    return GENGA_KICK_OK;
}

extern "C" const char* genga_kick_strerror(int code)
{
    switch (code) {
    case GENGA_KICK_OK: return "ok";
    case GENGA_KICK_E_NULL: return "a required pointer is NULL";
    case GENGA_KICK_E_ALIGN: return "a device pointer is not 16-byte aligned";
    case GENGA_KICK_E_SIZE: return "a size is out of range";
    case GENGA_KICK_E_LEVEL: return "changeover_level is outside [0, max_level]";
    case GENGA_KICK_E_CUDA: return "a CUDA call failed";
    case GENGA_KICK_E_NOMEM: return "host allocation failed";
    case -7: return "N exceeds GENGA_KICK_STATIC_MAX_BODIES (65536): the static scratch of genga_kick_list_static cannot hold it";   // genga_kick_static.h
    default: return "unknown genga_kick error code";
    }
}
