// C ABI of the close-encounter detection and of the multi-level step (include/genga_senc.h).  Host side only: the
// recursion SEnc of App. A as a fixed launch sequence over the library's own entry points.
#include "../../include/genga_senc.h"
#include "../../include/genga_bs.h"
#include "../../include/genga_group.h"
#include "../../include/genga_step.h"
#include "genga_kick_ctx.h"
#include "genga_senc_kernels.cuh"

#include <algorithm>

#define GENGA_SENC_MAX_LEVELS 4      // = GENGA_BS_MAX_LEVELS (rows of r_crit the Bulirsch-Stoer kernels take)

extern "C" int genga_detect(genga_kick_ctx* ctx, const double* pos0, const double* vel0, const double* pos1,
                            const double* vel1, const double* rcrit_row, double enc_factor, double h,
                            const int32_t* in_pairs, const int32_t* in_n_pairs, int64_t in_pair_rows, int32_t* out_pairs,
                            int32_t* out_npairs)
{
    if (!ctx || !pos0 || !vel0 || !pos1 || !vel1 || !rcrit_row || !in_n_pairs || !out_npairs) return GENGA_KICK_E_NULL;
    if (!out_pairs && ctx->cfg.pair_capacity > 0) return GENGA_KICK_E_NULL;
    if (!in_pairs && in_pair_rows > 0) return GENGA_KICK_E_NULL;
    if (genga_misaligned(pos0) || genga_misaligned(vel0) || genga_misaligned(pos1) || genga_misaligned(vel1) ||
        genga_misaligned(rcrit_row) || genga_misaligned(in_pairs) || genga_misaligned(out_pairs) ||
        genga_misaligned(out_npairs))
        return GENGA_KICK_E_ALIGN;
    if (in_pair_rows < 0 || !(enc_factor > 0.0)) return GENGA_KICK_E_SIZE;
    const long long N = ctx->N;
    cudaStream_t st = ctx->stream;
    GK_CUDA(ctx, cudaMemsetAsync(out_npairs, 0, ((size_t)N + 1) * sizeof(int32_t), st));
    const int blocks = (int)std::min<int64_t>(
        std::max<int64_t>((in_pair_rows + GENGA_SENC_THREADS - 1) / GENGA_SENC_THREADS, 1), 8 * ctx->num_sms);
    genga::detect_kernel<<<blocks, GENGA_SENC_THREADS, 0, st>>>(
        pos0, vel0, pos1, vel1, rcrit_row, enc_factor, h, N, reinterpret_cast<const int2*>(in_pairs), in_n_pairs,
        in_pair_rows, reinterpret_cast<int2*>(out_pairs), ctx->cfg.pair_capacity, out_npairs, ctx->status);
    GK_CUDA(ctx, cudaGetLastError());
    ctx->launches++;
    return GENGA_KICK_OK;
}

namespace {

// Library-owned scratch of one symplectic level (a slice of ctx->senc_slab)
struct Level {
    int32_t* cand;  int32_t* cand_np;     // pre-check output of the level's KickS: [cap][2], [N + 1]
    int32_t* enc;   int32_t* enc_np;      // detection output
    int32_t* group_of; int32_t* members; int32_t* offsets; int32_t* summary;
    double*  q0;    double* v0;           // state of the level's bodies before its drift
};

struct Senc {
    genga_kick_ctx* ctx;
    const genga_senc_config* cfg;
    double* pos; double* vel; const double* mass;
    double m_star, dt;
    double* rc;                           // [slevels][N]
    Level lv[GENGA_SENC_MAX_LEVELS];
    int32_t* stats;                       // [slevels][4] or null
    long long N, cap;
};

size_t up16(size_t b) { return (b + 15) & ~size_t(15); }

int copy_list(Senc& s, double* dq, double* dv, const double* sq, const double* sv, const int32_t* list,
              const int32_t* n_list)
{
    const int blocks = (int)std::min<long long>((s.N + GENGA_SENC_THREADS - 1) / GENGA_SENC_THREADS, 4LL * s.ctx->num_sms);
    genga::copy_list_kernel<<<blocks, GENGA_SENC_THREADS, 0, s.ctx->stream>>>(dq, dv, sq, sv, s.N, list, n_list, s.N);
    GK_CUDA(s.ctx, cudaGetLastError());
    s.ctx->launches++;
    return GENGA_KICK_OK;
}

// detection (or not) + grouping of the candidates of `level`; *enc / *n_enc: the close-encounter list of the level
int encounters(Senc& s, int level, double h, const int32_t** enc, const int32_t** n_enc)
{
    Level& L = s.lv[level];
    int rc;
    if (s.cfg->detect) {
        rc = genga_detect(s.ctx, L.q0, L.v0, s.pos, s.vel, s.rc + (size_t)level * s.N, 1.0, h, L.cand, L.cand_np + s.N,
                          s.cap, L.enc, L.enc_np);
        if (rc != GENGA_KICK_OK) return rc;
        *enc = L.enc; *n_enc = L.enc_np + s.N;
    } else {
        *enc = L.cand; *n_enc = L.cand_np + s.N;
    }
    rc = genga_group(s.ctx, *enc, *n_enc, s.cap, L.group_of, L.members, L.offsets, L.summary);
    if (rc != GENGA_KICK_OK) return rc;
    genga::senc_stats_kernel<<<1, 32, 0, s.ctx->stream>>>(s.stats ? s.stats + 4 * level : nullptr, L.cand_np + s.N, *n_enc,
                                                         L.summary, level == s.cfg->slevels - 1 ? 1 : 0, s.cap,
                                                         s.ctx->status);
    GK_CUDA(s.ctx, cudaGetLastError());
    s.ctx->launches++;
    return GENGA_KICK_OK;
}

// what follows the detection at `level`: the next level's sub-steps, or Bulirsch-Stoer at the deepest level
int senc(Senc& s, int level, const int32_t* pairs_up, const int32_t* n_up, const int32_t* bodies, const int32_t* n_bodies);

int descend(Senc& s, int level, double h, const int32_t* enc, const int32_t* n_enc)
{
    Level& L = s.lv[level];
    if (level < s.cfg->slevels - 1) {
        int rc = copy_list(s, s.pos, s.vel, L.q0, L.v0, L.members, L.summary + 1);      // restart before the drift
        if (rc != GENGA_KICK_OK) return rc;
        return senc(s, level + 1, enc, n_enc, L.members, L.summary + 1);
    }
    return genga_bs(s.ctx, L.q0, L.v0, s.mass, s.rc, level + 1, s.m_star, h, s.cfg->tol, L.members, L.offsets, L.summary,
                    s.pos, s.vel);
}

int senc(Senc& s, int level, const int32_t* pairs_up, const int32_t* n_up, const int32_t* bodies, const int32_t* n_bodies)
{
    Level& L = s.lv[level];
    double h = s.dt;
    for (int k = 0; k < level; k++) h /= (double)s.cfg->substeps;                       // dt / ds
    double* row = s.rc + (size_t)level * s.N;
    for (int sub = 0; sub < s.cfg->substeps; sub++) {
        int rc = genga_rcrit_list(s.ctx, s.pos, s.vel, s.mass, s.m_star, h, 2.0, 1, s.cfg->n1, s.cfg->n2, bodies,
                                  n_bodies, s.N, row);                                  // RcritS
        if (rc != GENGA_KICK_OK) return rc;
        rc = genga_kick_list(s.ctx, s.pos, s.vel, s.mass, s.rc, level, 0.5 * h, pairs_up, n_up, s.cap, nullptr, L.cand,
                             L.cand_np);                                                // KickS(dt/ds/2) + pre-check
        if (rc != GENGA_KICK_OK) return rc;
        rc = copy_list(s, L.q0, L.v0, s.pos, s.vel, bodies, n_bodies);
        if (rc != GENGA_KICK_OK) return rc;
        rc = genga_fg_list(s.ctx, s.pos, s.vel, s.m_star, h, bodies, n_bodies, s.N);    // FGS(dt/ds)
        if (rc != GENGA_KICK_OK) return rc;
        const int32_t *enc, *n_enc;
        rc = encounters(s, level, h, &enc, &n_enc);
        if (rc != GENGA_KICK_OK) return rc;
        rc = descend(s, level, h, enc, n_enc);
        if (rc != GENGA_KICK_OK) return rc;
        // the closing KickS writes its (unused) pre-check output over the level's candidate list
        rc = genga_kick_list(s.ctx, s.pos, s.vel, s.mass, s.rc, level, 0.5 * h, pairs_up, n_up, s.cap, nullptr, L.cand,
                             L.cand_np);                                                // KickS(dt/ds/2)
        if (rc != GENGA_KICK_OK) return rc;
    }
    return GENGA_KICK_OK;
}

}  // namespace

namespace {

int check_ml_args(genga_kick_ctx* ctx, double* pos, double* vel, const double* mass, double m_star,
                  const genga_senc_config* cfg, double* out_acc, int32_t* out_pairs, int32_t* out_npairs,
                  int32_t* out_stats, int min_levels)
{
    if (!ctx || !pos || !vel || !mass || !cfg || !out_npairs) return GENGA_KICK_E_NULL;
    if (!out_pairs && ctx->cfg.pair_capacity > 0) return GENGA_KICK_E_NULL;
    if (genga_misaligned(pos) || genga_misaligned(vel) || genga_misaligned(mass) || genga_misaligned(out_acc) ||
        genga_misaligned(out_pairs) || genga_misaligned(out_npairs) || genga_misaligned(out_stats))
        return GENGA_KICK_E_ALIGN;
    if (cfg->slevels < min_levels || cfg->slevels > GENGA_SENC_MAX_LEVELS || (cfg->slevels > 1 && cfg->substeps < 1) ||
        (cfg->slevels >= 1 && !(cfg->tol > 0.0)) || !(m_star > 0.0))
        return GENGA_KICK_E_SIZE;
    if (cfg->slevels - 1 > ctx->cfg.max_level) return GENGA_KICK_E_LEVEL;
    return GENGA_KICK_OK;
}

// cuts the library's slab for cfg->slevels levels (at least one r_crit row) plus one spare r_crit row (*rc_spare)
int setup_senc(genga_kick_ctx* ctx, double* pos, double* vel, const double* mass, double m_star, double dt,
               const genga_senc_config* cfg, int32_t* out_pairs, int32_t* out_npairs, int32_t* out_stats, Senc& s,
               double** rc_spare)
{
    const size_t N = (size_t)ctx->N, cap = (size_t)ctx->cfg.pair_capacity;
    const int SL = std::max(cfg->slevels, 1);
    cudaStream_t st = ctx->stream;
    // scratch: one slab, cut per level (kept for the next call with as many or fewer levels)
    const size_t b_pairs = up16(std::max<size_t>(cap, 1) * 2 * sizeof(int32_t)), b_np = up16((N + 1) * sizeof(int32_t));
    const size_t b_n = up16(N * sizeof(int32_t)), b_state = up16(3 * N * sizeof(double)), b_row = up16(N * sizeof(double));
    const size_t per_level = 2 * b_pairs + 2 * b_np + 2 * b_n + b_np + 16 + 2 * b_state;
    if (!ctx->senc_slab || ctx->senc_levels < SL) {
        if (ctx->senc_slab) { GK_CUDA(ctx, cudaStreamSynchronize(st)); cudaFree(ctx->senc_slab); ctx->senc_slab = nullptr; }
        GK_CUDA(ctx, cudaMalloc(&ctx->senc_slab, SL * (per_level + b_row) + b_row));
        ctx->senc_levels = SL;
    }
    s = Senc{};
    s.ctx = ctx; s.cfg = cfg; s.pos = pos; s.vel = vel; s.mass = mass; s.m_star = m_star; s.dt = dt;
    s.N = (long long)N; s.cap = (long long)cap; s.stats = out_stats;
    char* p = static_cast<char*>(ctx->senc_slab);
    *rc_spare = reinterpret_cast<double*>(p); p += b_row;
    s.rc = reinterpret_cast<double*>(p); p += SL * b_row;
    for (int l = 0; l < SL; l++) {
        Level& L = s.lv[l];
        L.cand = reinterpret_cast<int32_t*>(p); p += b_pairs;
        L.enc = reinterpret_cast<int32_t*>(p); p += b_pairs;
        L.cand_np = reinterpret_cast<int32_t*>(p); p += b_np;
        L.enc_np = reinterpret_cast<int32_t*>(p); p += b_np;
        L.group_of = reinterpret_cast<int32_t*>(p); p += b_n;
        L.members = reinterpret_cast<int32_t*>(p); p += b_n;
        L.offsets = reinterpret_cast<int32_t*>(p); p += b_np;
        L.summary = reinterpret_cast<int32_t*>(p); p += 16;
        L.q0 = reinterpret_cast<double*>(p); p += b_state;
        L.v0 = reinterpret_cast<double*>(p); p += b_state;
    }
    // level 0 writes its candidates where the caller reads them
    s.lv[0].cand = out_pairs; s.lv[0].cand_np = out_npairs;
    if (out_stats && cfg->slevels >= 1)
        GK_CUDA(ctx, cudaMemsetAsync(out_stats, 0, (size_t)cfg->slevels * 4 * sizeof(int32_t), st));
    return GENGA_KICK_OK;
}

// what lies between the two kicks of a step: HC(dt/2); FG(dt); detection, SEnc or grouping + Bulirsch-Stoer; HC(dt/2)
// (slevels == 0: no encounter branch -- genga_drift)
int middle(Senc& s)
{
    genga_kick_ctx* ctx = s.ctx;
    const size_t N = (size_t)s.N;
    if (s.cfg->slevels == 0) return genga_drift(ctx, s.pos, s.vel, s.mass, s.m_star, s.dt);
    int rc = genga_hc(ctx, s.pos, s.vel, s.mass, s.m_star, 0.5 * s.dt);
    if (rc != GENGA_KICK_OK) return rc;
    GK_CUDA(ctx, cudaMemcpyAsync(s.lv[0].q0, s.pos, 3 * N * sizeof(double), cudaMemcpyDeviceToDevice, ctx->stream));
    GK_CUDA(ctx, cudaMemcpyAsync(s.lv[0].v0, s.vel, 3 * N * sizeof(double), cudaMemcpyDeviceToDevice, ctx->stream));
    rc = genga_fg(ctx, s.pos, s.vel, s.m_star, s.dt);
    if (rc != GENGA_KICK_OK) return rc;
    const int32_t *enc, *n_enc;
    rc = encounters(s, 0, s.dt, &enc, &n_enc);
    if (rc != GENGA_KICK_OK) return rc;
    rc = descend(s, 0, s.dt, enc, n_enc);
    if (rc != GENGA_KICK_OK) return rc;
    return genga_hc(ctx, s.pos, s.vel, s.mass, s.m_star, 0.5 * s.dt);
}

}  // namespace

extern "C" int genga_multilevel_step(genga_kick_ctx* ctx, double* pos, double* vel, const double* mass, double m_star,
                                     double dt, const genga_senc_config* cfg, double* out_acc, int32_t* out_pairs,
                                     int32_t* out_npairs, int32_t* out_stats)
{
    int rc = check_ml_args(ctx, pos, vel, mass, m_star, cfg, out_acc, out_pairs, out_npairs, out_stats, 1);
    if (rc != GENGA_KICK_OK) return rc;
    Senc s;
    double* spare;
    rc = setup_senc(ctx, pos, vel, mass, m_star, dt, cfg, out_pairs, out_npairs, out_stats, s, &spare);
    if (rc != GENGA_KICK_OK) return rc;
    rc = genga_rcrit(ctx, pos, vel, mass, m_star, dt, 2.0, 1, cfg->n1, cfg->n2, s.rc);
    if (rc != GENGA_KICK_OK) return rc;
    rc = genga_kick(ctx, pos, vel, mass, s.rc, 0, 0.5 * dt, nullptr, out_pairs, out_npairs);
    if (rc != GENGA_KICK_OK) return rc;
    rc = middle(s);
    if (rc != GENGA_KICK_OK) return rc;
    return genga_kick_impl(ctx, pos, vel, mass, s.rc, 0, 0.5 * dt, out_acc, nullptr, nullptr);
}

extern "C" int genga_steps(genga_kick_ctx* ctx, double* pos, double* vel, const double* mass, double m_star, double dt,
                           int32_t n_steps, const genga_senc_config* cfg, double* out_acc, int32_t* out_pairs,
                           int32_t* out_npairs, int32_t* out_stats)
{
    int rc = check_ml_args(ctx, pos, vel, mass, m_star, cfg, out_acc, out_pairs, out_npairs, out_stats, 0);
    if (rc != GENGA_KICK_OK) return rc;
    if (n_steps < 1) return GENGA_KICK_E_SIZE;
    Senc s;
    double* spare;
    rc = setup_senc(ctx, pos, vel, mass, m_star, dt, cfg, out_pairs, out_npairs, out_stats, s, &spare);
    if (rc != GENGA_KICK_OK) return rc;
    const size_t N = (size_t)ctx->N;
    rc = genga_rcrit(ctx, pos, vel, mass, m_star, dt, 2.0, 1, cfg->n1, cfg->n2, s.rc);
    if (rc != GENGA_KICK_OK) return rc;
    rc = genga_kick(ctx, pos, vel, mass, s.rc, 0, 0.5 * dt, nullptr, out_pairs, out_npairs);
    if (rc != GENGA_KICK_OK) return rc;
    for (int step = 0; step < n_steps; step++) {
        rc = middle(s);
        if (rc != GENGA_KICK_OK) return rc;
        if (step == n_steps - 1) break;
        // closing kick of this step + Rcrit + opening kick and pre-check of the next: one pass over the pairs
        rc = genga_kick_merged_impl(ctx, pos, vel, mass, s.rc, spare, m_star, dt, cfg->n1, cfg->n2, nullptr, out_pairs,
                                    out_npairs);
        if (rc != GENGA_KICK_OK) return rc;
        GK_CUDA(ctx, cudaMemcpyAsync(s.rc, spare, N * sizeof(double), cudaMemcpyDeviceToDevice, ctx->stream));
    }
    return genga_kick_impl(ctx, pos, vel, mass, s.rc, 0, 0.5 * dt, out_acc, nullptr, nullptr);
}
