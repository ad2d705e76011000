// C ABI of the B200-native GENGA kick + close-encounter pre-check (include/genga_kick.h).
// Host side only: argument checks, scratch ownership, kernel launches on the caller's stream.
// Every step of the path runs in the kernels of genga_kick_kernels.cuh; there is no CPU fallback.
#include "genga_kick_ctx.h"
#include "../../include/genga_step.h"
#include "genga_kick_variants.h"
#include "genga_kick_kernels.cuh"
#include "genga_kick_sym.cuh"
#include "genga_kick_sort.cuh"

#include <algorithm>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

namespace {

int cuda_fail(genga_kick_ctx* ctx, cudaError_t e) { return genga_cuda_fail(ctx, e); }
bool misaligned(const void* p) { return genga_misaligned(p); }

template <int THREADS, int IPT, int JT, int CTAS>
cudaError_t launch_kick(const genga::KickParams& kp, cudaStream_t st)
{
    genga::kick_kernel<THREADS, IPT, JT, CTAS, GENGA_STAGES><<<kp.n_ctas, THREADS, 0, st>>>(kp);
    return cudaGetLastError();
}

// the compiled shapes: must list every entry of GENGA_VARIANTS
cudaError_t dispatch_kick(const genga_kick_plan& pl, const genga::KickParams& kp, cudaStream_t st)
{
#define GK_SHAPE(T, I, J, C)                                                          \
    if (pl.threads == T && pl.i_per_thread == I && pl.j_tile == J)                    \
        return launch_kick<T, I, J, C>(kp, st);
    GK_SHAPE(256, 2, 256, 2)
    GK_SHAPE(128, 2, 128, 4)
    GK_SHAPE(128, 1, 64, 4)
#undef GK_SHAPE
    return cudaErrorInvalidConfiguration;
}

}  // namespace

extern "C" int genga_kick_init(const genga_kick_config* cfg, genga_kick_ctx** out_ctx)
{
    if (!cfg || !out_ctx) return GENGA_KICK_E_NULL;
    const int64_t N = (int64_t)cfg->n_massive + (int64_t)cfg->n_test;
    if (cfg->n_massive < 0 || cfg->n_test < 0 || N <= 0 || N > GENGA_MAX_BODIES || cfg->pair_capacity < 0)
        return GENGA_KICK_E_SIZE;
    if (cfg->max_level < 0 || cfg->max_level > 62) return GENGA_KICK_E_LEVEL;
    if (cfg->order_mode < GENGA_KICK_ORDER_AUTO || cfg->order_mode > GENGA_KICK_ORDER_SORTED) return GENGA_KICK_E_SIZE;
    if (cfg->tp_mode < 0 || cfg->tp_mode > 2) return GENGA_KICK_E_SIZE;

    genga_kick_ctx* ctx = new (std::nothrow) genga_kick_ctx();
    if (!ctx) return GENGA_KICK_E_NOMEM;
    ctx->cfg = *cfg;
    ctx->N = N;
    ctx->stream = nullptr;
    ctx->launches = 0;

    int rc = GENGA_KICK_OK;
    cudaError_t e;
    int ndev = 0;
    cudaDeviceProp prop;
    if ((e = cudaGetDeviceCount(&ndev)) != cudaSuccess) goto cuda_error;
    if (cfg->device < 0 || cfg->device >= ndev) { e = cudaErrorInvalidDevice; goto cuda_error; }
    if ((e = cudaSetDevice(cfg->device)) != cudaSuccess) goto cuda_error;
    if ((e = cudaGetDeviceProperties(&prop, cfg->device)) != cudaSuccess) goto cuda_error;
    if (prop.major != 10) { e = cudaErrorNoKernelImageForDevice; goto cuda_error; }   // sm_100a only
    ctx->num_sms = prop.multiProcessorCount;

    ctx->plans = static_cast<genga_kick_plan*>(std::calloc((size_t)cfg->max_level + 1, sizeof(genga_kick_plan)));
    if (!ctx->plans) { rc = GENGA_KICK_E_NOMEM; goto fail; }
    {
        int64_t max_partial = 1;
        for (int l = 0; l <= cfg->max_level; l++) {
            rc = genga_kick_make_plan(cfg->n_massive, cfg->n_test, l, ctx->num_sms, &ctx->plans[l]);
            if (rc != GENGA_KICK_OK) goto fail;
            if (ctx->plans[l].partial_doubles > max_partial) max_partial = ctx->plans[l].partial_doubles;
        }
        const int64_t nr = ctx->plans[0].n_rec;
        ctx->n_rec_alloc = nr;
        if ((e = cudaMalloc(&ctx->rxy, (size_t)nr * sizeof(double2))) != cudaSuccess) goto cuda_error;
        if ((e = cudaMalloc(&ctx->rzm, (size_t)nr * sizeof(double2))) != cudaSuccess) goto cuda_error;
        if ((e = cudaMalloc(&ctx->rfw, (size_t)nr * sizeof(int))) != cudaSuccess) goto cuda_error;
        if ((e = cudaMalloc(&ctx->rfw_ref, (size_t)nr * sizeof(int))) != cudaSuccess) goto cuda_error;
        if ((e = cudaMalloc(&ctx->need_near, ((size_t)cfg->max_level + 1) * sizeof(int))) != cudaSuccess) goto cuda_error;
        if ((e = cudaMemset(ctx->need_near, 0, ((size_t)cfg->max_level + 1) * sizeof(int))) != cudaSuccess) goto cuda_error;
        if ((e = cudaMalloc(&ctx->ridx, (size_t)nr * sizeof(int))) != cudaSuccess) goto cuda_error;
        if ((e = cudaMalloc(&ctx->cblo, (size_t)(nr / GENGA_GROUP) * sizeof(float4))) != cudaSuccess) goto cuda_error;
        if ((e = cudaMalloc(&ctx->cbhi, (size_t)(nr / GENGA_GROUP) * sizeof(float4))) != cudaSuccess) goto cuda_error;
        ctx->sorted = cfg->order_mode == GENGA_KICK_ORDER_SORTED ||
                      (cfg->order_mode == GENGA_KICK_ORDER_AUTO && N >= GENGA_SORT_MIN_BODIES);
        if (ctx->sorted) {
            ctx->sort_blocks = (int)((N + genga::genga_sort_block(N) - 1) / genga::genga_sort_block(N));
            const size_t nc = (size_t)GENGA_SORT_MAXDIGITS * ctx->sort_blocks;
            if ((e = cudaMalloc(&ctx->bbox, 4 * sizeof(unsigned))) != cudaSuccess) goto cuda_error;
            if ((e = cudaMalloc(&ctx->keys_a, (size_t)N * sizeof(unsigned))) != cudaSuccess) goto cuda_error;
            if ((e = cudaMalloc(&ctx->keys_b, (size_t)N * sizeof(unsigned))) != cudaSuccess) goto cuda_error;
            if ((e = cudaMalloc(&ctx->vals_a, (size_t)N * sizeof(int))) != cudaSuccess) goto cuda_error;
            if ((e = cudaMalloc(&ctx->vals_b, (size_t)N * sizeof(int))) != cudaSuccess) goto cuda_error;
            if ((e = cudaMalloc(&ctx->counts, nc * sizeof(int))) != cudaSuccess) goto cuda_error;
        }
        rc = genga_kick_make_plan_sym(cfg->n_massive, cfg->n_test, ctx->num_sms, &ctx->plan_sym);
        if (rc != GENGA_KICK_OK) goto fail;
        if (ctx->plan_sym.n_ctas > 0) {
            if ((e = cudaMalloc(&ctx->partial_sym, (size_t)ctx->plan_sym.partial_doubles * sizeof(double))) != cudaSuccess) goto cuda_error;
            if ((e = cudaMalloc(&ctx->react, (size_t)ctx->plan_sym.react_doubles * sizeof(double))) != cudaSuccess) goto cuda_error;
            {
                std::vector<int64_t> tab((size_t)ctx->plan_sym.n_ctas + 1, 0);
                rc = genga_kick_plan_sym_table(&ctx->plan_sym, tab.data());
                if (rc != GENGA_KICK_OK) goto fail;
                if ((e = cudaMalloc(&ctx->sym_t0, tab.size() * sizeof(long long))) != cudaSuccess) goto cuda_error;
                if ((e = cudaMemcpy(ctx->sym_t0, tab.data(), tab.size() * sizeof(long long), cudaMemcpyHostToDevice)) != cudaSuccess) goto cuda_error;
            }
            if (cfg->n_test > 0) {
                rc = genga_kick_make_plan_tprows(cfg->n_massive, cfg->n_test, ctx->num_sms, &ctx->plan_tprows);
                if (rc != GENGA_KICK_OK) goto fail;
                if (ctx->plan_tprows.partial_doubles > max_partial) max_partial = ctx->plan_tprows.partial_doubles;
            }
        }
        if ((e = cudaMalloc(&ctx->partial, (size_t)max_partial * sizeof(double))) != cudaSuccess) goto cuda_error;
        ctx->tp2 = cfg->tp_mode == 2 && cfg->n_test > 0 && cfg->n_massive > 0;
        if (ctx->tp2) {
            rc = genga_kick_make_plan_tp2(cfg->n_massive, cfg->n_test, ctx->num_sms, &ctx->plan_tp2);
            if (rc != GENGA_KICK_OK) goto fail;
            if ((e = cudaMalloc(&ctx->partial2, (size_t)std::max<int64_t>(ctx->plan_tp2.partial_doubles, 1) * sizeof(double))) != cudaSuccess)
                goto cuda_error;
        }
        ctx->cand_capacity = std::min<int64_t>(std::max<int64_t>(GENGA_CAND_PER_BODY * N, GENGA_CAND_MIN), GENGA_CAND_MAX);
        if ((e = cudaMalloc(&ctx->cand, (size_t)ctx->cand_capacity * sizeof(int2))) != cudaSuccess) goto cuda_error;
        if ((e = cudaMalloc(&ctx->ncand, sizeof(int))) != cudaSuccess) goto cuda_error;
        if ((e = cudaMalloc(&ctx->fx, (size_t)nr * 3 * GENGA_FX_LIMBS * sizeof(unsigned long long))) != cudaSuccess) goto cuda_error;
        if ((e = cudaMemset(ctx->fx, 0, (size_t)nr * 3 * GENGA_FX_LIMBS * sizeof(unsigned long long))) != cudaSuccess) goto cuda_error;
        if ((e = cudaMalloc(&ctx->touched, (size_t)nr * sizeof(int))) != cudaSuccess) goto cuda_error;
        if ((e = cudaMemset(ctx->touched, 0, (size_t)nr * sizeof(int))) != cudaSuccess) goto cuda_error;
        if ((e = cudaMalloc(&ctx->status, sizeof(int))) != cudaSuccess) goto cuda_error;
        if ((e = cudaMemset(ctx->status, 0, sizeof(int))) != cudaSuccess) goto cuda_error;
    }
    *out_ctx = ctx;
    return GENGA_KICK_OK;

cuda_error:
    (void)e;                       // the context is freed below: the text of e cannot be kept
    rc = GENGA_KICK_E_CUDA;
fail:
    genga_kick_free(ctx);
    return rc;
}

extern "C" int genga_kick_set_stream(genga_kick_ctx* ctx, void* cuda_stream)
{
    if (!ctx) return GENGA_KICK_E_NULL;
    ctx->stream = static_cast<cudaStream_t>(cuda_stream);
    return GENGA_KICK_OK;
}

extern "C" int genga_kick_set_order_reuse(genga_kick_ctx* ctx, int32_t on)
{
    if (!ctx) return GENGA_KICK_E_NULL;
    if (on < 0 || on > GENGA_KICK_REUSE_LIST) return GENGA_KICK_E_SIZE;
    ctx->reuse_order = on != 0;
    ctx->reuse_list = on == GENGA_KICK_REUSE_LIST;
    return GENGA_KICK_OK;
}

extern "C" int genga_kick(genga_kick_ctx* ctx, const double* pos, double* vel, const double* mass, const double* rcrit,
                          int32_t changeover_level, double dt, double* out_acc, int32_t* out_pairs, int32_t* out_npairs)
{
    if (!out_npairs) return GENGA_KICK_E_NULL;
    return genga_kick_impl(ctx, pos, vel, mass, rcrit, changeover_level, dt, out_acc, out_pairs, out_npairs);
}

namespace {

// A kick in two halves.  kick_front: internal order, records, and the pair loop(s) -- the far-field partial sums and
// the candidate list of the pairs that tripped the filter (built from the rows of `rcrit`, the filter radius scaled
// by fw_scale).  kick_back: the exact path over that list with the rows of kp.rcrit (weights, pre-check, pair list)
// and the fixed-order sum -> out_acc, v += dt a.  One front can serve several backs (genga_kick_merged).
int kick_front(genga_kick_ctx* ctx, const double* pos, const double* mass, const double* rcrit, int32_t changeover_level,
               double fw_scale, int32_t* out_pairs, int32_t* out_npairs, genga::KickParams& kp);
int kick_back(genga_kick_ctx* ctx, const genga::KickParams& kp, int32_t changeover_level, double dt, double* out_acc,
              double* vel);

}  // namespace

int genga_kick_impl(genga_kick_ctx* ctx, const double* pos, double* vel, const double* mass, const double* rcrit,
                    int32_t changeover_level, double dt, double* out_acc, int32_t* out_pairs, int32_t* out_npairs)
{
    if (!ctx || !pos || !mass || !rcrit) return GENGA_KICK_E_NULL;
    if (!out_acc && !vel) return GENGA_KICK_E_NULL;
    if (!out_pairs && out_npairs && ctx->cfg.pair_capacity > 0) return GENGA_KICK_E_NULL;
    if (misaligned(pos) || misaligned(vel) || misaligned(mass) || misaligned(rcrit) || misaligned(out_acc) ||
        misaligned(out_pairs) || misaligned(out_npairs))
        return GENGA_KICK_E_ALIGN;
    if (changeover_level < 0 || changeover_level > ctx->cfg.max_level) return GENGA_KICK_E_LEVEL;
    genga::KickParams kp = {};
    int rc = kick_front(ctx, pos, mass, rcrit, changeover_level, 1.0, out_pairs, out_npairs, kp);
    if (rc != GENGA_KICK_OK) return rc;
    return kick_back(ctx, kp, changeover_level, dt, out_acc, vel);
}

namespace {

int kick_front(genga_kick_ctx* ctx, const double* pos, const double* mass, const double* rcrit, int32_t changeover_level,
               double fw_scale, int32_t* out_pairs, int32_t* out_npairs, genga::KickParams& kp)
{
    const genga_kick_plan& pl = ctx->plans[changeover_level];
    const int N = (int)ctx->N;
    const int n_rec = (int)pl.n_rec;
    cudaStream_t st = ctx->stream;

    if (ctx->sorted && !(ctx->reuse_order && ctx->order_valid)) {
        // stable LSD radix sort of the 17-bit keys: digits of 8 and 9 bits
        const int nb = ctx->sort_blocks, sb = genga::genga_sort_block(N);
        genga::sort_init_kernel<<<1, 32, 0, st>>>(ctx->bbox);
        genga::bbox_kernel<<<std::min((N + 255) / 256, 8 * ctx->num_sms), 256, 0, st>>>(pos, N, ctx->bbox);
        genga::key_hist_kernel<<<nb, GENGA_SORT_THREADS, 0, st>>>(pos, N, ctx->cfg.n_massive, ctx->bbox, ctx->keys_a,
                                                                  ctx->vals_a, 8, nb, ctx->counts, sb);
        genga::scan_kernel<<<1, 1024, 0, st>>>(ctx->counts, 256 * nb);
        genga::radix_scatter_kernel<<<nb, GENGA_SORT_THREADS, 0, st>>>(ctx->keys_a, ctx->vals_a, N, 0, 8, nb, ctx->counts,
                                                                       ctx->keys_b, ctx->vals_b, sb);
        genga::radix_hist_kernel<<<nb, GENGA_SORT_THREADS, 0, st>>>(ctx->keys_b, N, 8, 9, nb, ctx->counts, sb);
        genga::scan_kernel<<<1, 1024, 0, st>>>(ctx->counts, 512 * nb);
        genga::radix_scatter_kernel<<<nb, GENGA_SORT_THREADS, 0, st>>>(ctx->keys_b, ctx->vals_b, N, 8, 9, nb, ctx->counts,
                                                                       nullptr, ctx->vals_a, sb);
        GK_CUDA(ctx, cudaGetLastError());
        ctx->launches += 8;
        ctx->order_valid = true;
        ctx->list_valid = false;
    }
    // GENGA_KICK_REUSE_LIST: a level >= 1 kick evaluates the candidate list the level-0 kick has left
    const bool keep_list = changeover_level > 0 && ctx->reuse_list && ctx->list_valid;
    if (!keep_list) ctx->list_valid = changeover_level == 0;   // whose list ctx->cand holds after this call
    kp = genga::KickParams{};
    {
        kp.rxy = ctx->rxy; kp.rzm = ctx->rzm; kp.rfw = ctx->rfw; kp.ridx = ctx->ridx;
        kp.cblo = ctx->cblo; kp.cbhi = ctx->cbhi;
        kp.rcrit = rcrit;
        kp.N = N; kp.n_massive = ctx->cfg.n_massive; kp.L = changeover_level; kp.f = ctx->cfg.enc_factor;
        kp.react = ctx->tp2 && changeover_level > 0 ? 1 : 0; kp.j_rec0 = 0; kp.i_rec0 = 0; kp.force_only = 0; kp.i_rec_end = n_rec;
        kp.n_j_tiles = pl.n_j_tiles; kp.n_ctas = pl.n_ctas; kp.max_segs = pl.max_segs; kp.n_tiles = pl.n_tiles;
        kp.partial = ctx->partial;
        kp.out_pairs = out_pairs; kp.capacity = ctx->cfg.pair_capacity; kp.out_npairs = out_npairs;
        kp.status = ctx->status;
        kp.cand = ctx->cand; kp.cand_capacity = ctx->cand_capacity; kp.ncand = ctx->ncand;
        kp.fx = ctx->fx; kp.fx_stride = ctx->n_rec_alloc; kp.touched = ctx->touched;
        kp.need_near = keep_list ? ctx->need_near + changeover_level : nullptr;
    }
    {
        const int blocks = (int)((std::max<int64_t>(n_rec, N + 1) + 255) / 256);
        genga::pack_kernel<<<blocks, 256, 0, st>>>(pos, mass, rcrit, ctx->sorted ? ctx->vals_a : nullptr, N,
                                                   ctx->cfg.n_massive, pl.m_pad, n_rec, changeover_level, ctx->cfg.G,
                                                   ctx->cfg.enc_factor, fw_scale, ctx->rxy, ctx->rzm, ctx->rfw, ctx->ridx,
                                                   ctx->cblo, ctx->cbhi, out_npairs, ctx->ncand,
                                                   ctx->rfw_ref, ctx->need_near,
                                                   ctx->cfg.max_level + 1, keep_list ? 1 : 0);
        GK_CUDA(ctx, cudaGetLastError());
        ctx->launches++;
    }
    const bool use_sym = changeover_level == 0 && ctx->plan_sym.n_ctas > 0;
    if (pl.n_ctas > 0) {
        if (ctx->timing) GK_CUDA(ctx, cudaEventRecord(ctx->ev[2 * changeover_level], st));
        if (changeover_level == 0 && use_sym) {
            // massive x massive: every unordered pair once (kick_sym_kernel); the particles' rows one-sided beside it
            const genga_kick_plan& ps = ctx->plan_sym;
            genga::KickParams ks = kp;
            ks.n_j_tiles = ps.n_j_tiles; ks.n_ctas = ps.n_ctas; ks.max_segs = ps.max_segs; ks.n_tiles = ps.n_tiles;
            ks.partial = ctx->partial_sym;
            ks.i_rec_end = (ctx->cfg.n_massive + 31) / 32 * 32;
            genga::SymParams sp = {ps.n_i_blocks, ps.tiles_per_iblock, ctx->react, ctx->sym_t0};
            genga::kick_sym_kernel<GENGA_SYM_THREADS, GENGA_SYM_IPT, GENGA_STAGES><<<ps.n_ctas, GENGA_SYM_THREADS, 0, st>>>(ks, sp);
            GK_CUDA(ctx, cudaGetLastError());
            if (ctx->plan_tprows.n_ctas > 0) {
                const genga_kick_plan& pt = ctx->plan_tprows;
                genga::KickParams kt = kp;
                kt.n_j_tiles = pt.n_j_tiles; kt.n_ctas = pt.n_ctas; kt.max_segs = pt.max_segs; kt.n_tiles = pt.n_tiles;
                kt.i_rec0 = pl.m_pad;
                GK_CUDA(ctx, dispatch_kick(pt, kt, st));
                ctx->launches++;
            }
        } else if (changeover_level == 0) {
            GK_CUDA(ctx, dispatch_kick(pl, kp, st));
        } else if (!keep_list) {
            // W_L = 0 exactly outside the filter radius: a neighbour search, no tile decomposition
            const int n_igroups = n_rec / GENGA_GROUP, wpc = GENGA_NEAR_THREADS / 32;
            const int n_jgroups = pl.m_pad / GENGA_GROUP;
            const int jsplit = n_jgroups >= 8 * GENGA_NEAR_JSPLIT ? GENGA_NEAR_JSPLIT : 1;
            const int ichunks = (n_igroups + wpc - 1) / wpc;
            genga::near_kernel<false><<<dim3(ichunks, jsplit), GENGA_NEAR_THREADS, 0, st>>>(kp, n_rec, 0, n_jgroups, 0);
            GK_CUDA(ctx, cudaGetLastError());
        }
        if (ctx->timing) {
            GK_CUDA(ctx, cudaEventRecord(ctx->ev[2 * changeover_level + 1], st));
            ctx->ev_set[changeover_level] = true;
        }
        if (!keep_list) ctx->launches++;
        if (ctx->tp2 && changeover_level == 0 && ctx->plan_tp2.n_ctas > 0) {
            // TP 2, far field of the massive bodies' sum over the semi-active particles (at level >= 1 it is 0)
            const genga_kick_plan& p2 = ctx->plan_tp2;
            genga::KickParams k2 = kp;
            k2.n_j_tiles = p2.n_j_tiles; k2.n_ctas = p2.n_ctas; k2.max_segs = p2.max_segs; k2.n_tiles = p2.n_tiles;
            k2.partial = ctx->partial2; k2.j_rec0 = pl.m_pad; k2.force_only = 1; k2.i_rec_end = pl.m_pad;
            GK_CUDA(ctx, dispatch_kick(p2, k2, st));
            ctx->launches++;
        }
    }
    return GENGA_KICK_OK;
}

int kick_back(genga_kick_ctx* ctx, const genga::KickParams& kp, int32_t changeover_level, double dt, double* out_acc,
              double* vel)
{
    const genga_kick_plan& pl = ctx->plans[changeover_level];
    const int N = (int)ctx->N;
    const int n_rec = (int)pl.n_rec;
    cudaStream_t st = ctx->stream;
    const bool use_sym = changeover_level == 0 && ctx->plan_sym.n_ctas > 0;
    if (pl.n_ctas > 0) {
        {
            // fallback for an overflowed candidate list: returns at once otherwise (see near_kernel<true>)
            const int wpc = GENGA_NEAR_THREADS / 32;
            genga::near_kernel<true><<<(n_rec / GENGA_GROUP + wpc - 1) / wpc, GENGA_NEAR_THREADS, 0, st>>>(
                kp, n_rec, 0, pl.m_pad / GENGA_GROUP, 0);
            if (ctx->tp2 && changeover_level == 0)
                genga::near_kernel<true><<<(pl.m_pad / GENGA_GROUP + wpc - 1) / wpc, GENGA_NEAR_THREADS, 0, st>>>(
                    kp, pl.m_pad, pl.m_pad / GENGA_GROUP, (n_rec - pl.m_pad) / GENGA_GROUP, 1);
            ctx->launches += ctx->tp2 && changeover_level == 0 ? 2 : 1;
        }
        // exact path: CTAs walk the list the pair loop has written in rounds of 1024 candidates
        genga::exact_kernel<<<4 * ctx->num_sms, 256, 0, st>>>(kp);
        GK_CUDA(ctx, cudaGetLastError());
        ctx->launches++;
    }
    {
        // level >= 1: no partial segments (n_ctas = 0), every term comes from the exact path
        auto seg_of = [](const genga_kick_plan& q, const double* partial, int rec0, int rec_end, bool on) {
            genga::SegPlan sg = {};
            sg.partial = partial; sg.IB = q.i_block > 0 ? q.i_block : 1; sg.n_j_tiles = q.n_j_tiles > 0 ? q.n_j_tiles : 1;
            sg.n_ctas = on ? q.n_ctas : 0; sg.max_segs = q.max_segs; sg.n_tiles = q.n_tiles > 0 ? q.n_tiles : 1;
            sg.rec0 = rec0; sg.rec_end = rec_end;
            sg.symmetric = q.symmetric; sg.r = q.tiles_per_iblock; sg.n_rows = q.n_i_blocks;
            return sg;
        };
        const genga_kick_plan& p2 = ctx->plan_tp2;
        const bool second = ctx->tp2 && changeover_level == 0 && p2.n_ctas > 0;
        genga::ReduceParams rp = {};
        if (use_sym) {
            rp.seg[0] = seg_of(ctx->plan_sym, ctx->partial_sym, 0, pl.m_pad, true);
            rp.seg[0].tbegin = ctx->sym_t0;
            rp.react = ctx->react; rp.react_jt = ctx->plan_sym.j_tile;
            rp.seg[2] = seg_of(ctx->plan_tprows, ctx->partial, pl.m_pad, n_rec, ctx->plan_tprows.n_ctas > 0);
        } else {
            rp.seg[0] = seg_of(pl, ctx->partial, 0, n_rec, changeover_level == 0);
            rp.seg[2] = seg_of(pl, ctx->partial, 0, 0, false);
        }
        rp.seg[1] = seg_of(p2, ctx->partial2, 0, pl.m_pad, second);
        genga::reduce_kernel<<<(n_rec + GENGA_REDUCE_THREADS - 1) / GENGA_REDUCE_THREADS, GENGA_REDUCE_THREADS, 0, st>>>(
            rp, ctx->ridx, n_rec, N, dt, ctx->fx, ctx->n_rec_alloc, ctx->touched,
                                                                  ctx->status, out_acc, vel);
        GK_CUDA(ctx, cudaGetLastError());
        ctx->launches++;
    }
    return GENGA_KICK_OK;
}

}  // namespace

// The closing Kick(dt/2) of a step and the opening Kick(dt/2) + pre-check of the next act on the same positions
// (App. A PAPER.md:986-992 repeated): one pass over the pairs serves both.  They differ only in the critical radii --
// the next step's Rcrit(dt) is taken from the velocities AFTER the closing kick -- hence only in the pairs inside a
// critical radius, i.e. in the candidate list: far field once, exact path twice.
//     a_A = far + exact(rc_old);  v += (dt/2) a_A;  rc_new = Rcrit(pos, v);  a_B = far + exact(rc_new), pre-check;
//     v += (dt/2) a_B
// Equal to the two separate kicks up to the rounding of the far-field sum (whose filter radius is that of rc_old
// times 1 + GENGA_MERGE_MARGIN, so that the list also holds the pairs inside the new radii; a body whose critical
// radius grew by more raises GENGA_KICK_STATUS_RCRIT_JUMP: repeat those steps with genga_step).
int genga_kick_merged_impl(genga_kick_ctx* ctx, const double* pos, double* vel, const double* mass, const double* rc_old,
                           double* rc_new, double m_star, double dt_step, double n1, double n2, double* out_acc,
                           int32_t* out_pairs, int32_t* out_npairs)
{
    if (!ctx || !pos || !vel || !mass || !rc_old || !rc_new || !out_npairs) return GENGA_KICK_E_NULL;
    if (!out_pairs && ctx->cfg.pair_capacity > 0) return GENGA_KICK_E_NULL;
    if (misaligned(pos) || misaligned(vel) || misaligned(mass) || misaligned(rc_old) || misaligned(rc_new) ||
        misaligned(out_acc) || misaligned(out_pairs) || misaligned(out_npairs))
        return GENGA_KICK_E_ALIGN;
    genga::KickParams kp = {};
    int rc = kick_front(ctx, pos, mass, rc_old, 0, 1.0 + GENGA_MERGE_MARGIN, out_pairs, out_npairs, kp);
    if (rc != GENGA_KICK_OK) return rc;
    genga::KickParams ka = kp;                             // the closing kick: no pre-check output
    ka.out_pairs = nullptr; ka.out_npairs = nullptr;
    rc = kick_back(ctx, ka, 0, 0.5 * dt_step, nullptr, vel);
    if (rc != GENGA_KICK_OK) return rc;
    rc = genga_rcrit(ctx, pos, vel, mass, m_star, dt_step, 2.0, 1, n1, n2, rc_new);
    if (rc != GENGA_KICK_OK) return rc;
    const int N = (int)ctx->N;
    genga::rcrit_jump_kernel<<<(N + 255) / 256, 256, 0, ctx->stream>>>(rc_old, rc_new, N, 1.0 + GENGA_MERGE_MARGIN,
                                                                     ctx->status);
    GK_CUDA(ctx, cudaGetLastError());
    ctx->launches++;
    genga::KickParams kb = kp;                             // the opening kick of the next step
    kb.rcrit = rc_new;
    return kick_back(ctx, kb, 0, 0.5 * dt_step, out_acc, vel);
}

extern "C" int genga_kick_list(genga_kick_ctx* ctx, const double* pos, double* vel, const double* mass, const double* rcrit,
                               int32_t changeover_level, double dt, const int32_t* in_pairs, const int32_t* in_n_pairs,
                               int64_t in_pair_rows, double* out_acc, int32_t* out_pairs, int32_t* out_npairs)
{
    if (!ctx || !pos || !mass || !rcrit || !in_n_pairs || !out_npairs) return GENGA_KICK_E_NULL;
    if (!out_acc && !vel) return GENGA_KICK_E_NULL;
    if (!out_pairs && ctx->cfg.pair_capacity > 0) return GENGA_KICK_E_NULL;
    if (in_pair_rows < 0) return GENGA_KICK_E_SIZE;
    if (!in_pairs && in_pair_rows > 0) return GENGA_KICK_E_NULL;
    if (misaligned(pos) || misaligned(vel) || misaligned(mass) || misaligned(rcrit) || misaligned(out_acc) ||
        misaligned(out_pairs) || misaligned(out_npairs) || misaligned(in_pairs))
        return GENGA_KICK_E_ALIGN;
    if (changeover_level < 0 || changeover_level > ctx->cfg.max_level) return GENGA_KICK_E_LEVEL;
    const int N = (int)ctx->N;
    cudaStream_t st = ctx->stream;
    genga::KickParams kp = {};
    kp.rcrit = rcrit;
    kp.N = N; kp.n_massive = ctx->cfg.n_massive; kp.L = changeover_level; kp.f = ctx->cfg.enc_factor;
    kp.out_pairs = out_pairs; kp.capacity = ctx->cfg.pair_capacity; kp.out_npairs = out_npairs;
    kp.status = ctx->status;
    kp.fx = ctx->fx; kp.fx_stride = ctx->n_rec_alloc; kp.touched = ctx->touched;
    GK_CUDA(ctx, cudaMemsetAsync(out_npairs, 0, ((size_t)N + 1) * sizeof(int32_t), st));
    const int blocks = (int)std::min<int64_t>(std::max<int64_t>((in_pair_rows + 1023) / 1024, 1), 8 * ctx->num_sms);
    genga::list_kick_kernel<<<blocks, 256, 0, st>>>(kp, pos, mass, ctx->cfg.G, reinterpret_cast<const int2*>(in_pairs),
                                                    in_n_pairs, in_pair_rows, ctx->cfg.tp_mode == 2 ? 1 : 0);
    genga::list_reduce_kernel<<<(N + 255) / 256, 256, 0, st>>>(ctx->fx, ctx->n_rec_alloc, ctx->touched, N, dt, ctx->status, out_acc, vel);
    GK_CUDA(ctx, cudaGetLastError());
    ctx->launches += 2;
    return GENGA_KICK_OK;
}

namespace {
template <typename T>
int ensure(genga_kick_ctx* ctx, T** p, size_t count)
{
    if (*p) return GENGA_KICK_OK;
    GK_CUDA(ctx, cudaMalloc(p, count * sizeof(T) + 16));
    return GENGA_KICK_OK;
}
}  // namespace

extern "C" int genga_kick_host(genga_kick_ctx* ctx, const double* pos, double* vel, const double* mass,
                               const double* rcrit, int32_t changeover_level, double dt, double* out_acc,
                               int32_t* out_pairs, int32_t* out_npairs)
{
    if (!ctx || !pos || !mass || !rcrit || !out_npairs) return GENGA_KICK_E_NULL;
    if (!out_acc && !vel) return GENGA_KICK_E_NULL;
    if (changeover_level < 0 || changeover_level > ctx->cfg.max_level) return GENGA_KICK_E_LEVEL;
    const size_t N = (size_t)ctx->N;
    const size_t cap = (size_t)ctx->cfg.pair_capacity;
    const size_t rows = (size_t)ctx->cfg.max_level + 1;
    cudaStream_t st = ctx->stream;
    int rc;
    if ((rc = ensure(ctx, &ctx->h_pos, 3 * N))) return rc;
    if ((rc = ensure(ctx, &ctx->h_mass, N))) return rc;
    if ((rc = ensure(ctx, &ctx->h_rcrit, rows * N))) return rc;
    if ((rc = ensure(ctx, &ctx->h_acc, 3 * N))) return rc;
    if ((rc = ensure(ctx, &ctx->h_npairs, N + 1))) return rc;
    if ((rc = ensure(ctx, &ctx->h_pairs, 2 * cap + 4))) return rc;
    if (vel && (rc = ensure(ctx, &ctx->h_vel, 3 * N))) return rc;

    GK_CUDA(ctx, cudaMemcpyAsync(ctx->h_pos, pos, 3 * N * sizeof(double), cudaMemcpyHostToDevice, st));
    GK_CUDA(ctx, cudaMemcpyAsync(ctx->h_mass, mass, N * sizeof(double), cudaMemcpyHostToDevice, st));
    GK_CUDA(ctx, cudaMemcpyAsync(ctx->h_rcrit, rcrit, ((size_t)changeover_level + 1) * N * sizeof(double),
                                 cudaMemcpyHostToDevice, st));
    if (vel) GK_CUDA(ctx, cudaMemcpyAsync(ctx->h_vel, vel, 3 * N * sizeof(double), cudaMemcpyHostToDevice, st));

    rc = genga_kick(ctx, ctx->h_pos, vel ? ctx->h_vel : nullptr, ctx->h_mass, ctx->h_rcrit, changeover_level, dt,
                    ctx->h_acc, cap ? ctx->h_pairs : nullptr, ctx->h_npairs);
    if (rc != GENGA_KICK_OK) return rc;

    if (out_acc) GK_CUDA(ctx, cudaMemcpyAsync(out_acc, ctx->h_acc, 3 * N * sizeof(double), cudaMemcpyDeviceToHost, st));
    if (vel) GK_CUDA(ctx, cudaMemcpyAsync(vel, ctx->h_vel, 3 * N * sizeof(double), cudaMemcpyDeviceToHost, st));
    GK_CUDA(ctx, cudaMemcpyAsync(out_npairs, ctx->h_npairs, (N + 1) * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    GK_CUDA(ctx, cudaStreamSynchronize(st));
    if (out_pairs && cap) {
        size_t got = (size_t)out_npairs[N];
        if (got > cap) got = cap;
        if (got) GK_CUDA(ctx, cudaMemcpyAsync(out_pairs, ctx->h_pairs, 2 * got * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
        GK_CUDA(ctx, cudaStreamSynchronize(st));
    }
    return GENGA_KICK_OK;
}

extern "C" int genga_kick_get_plan(const genga_kick_ctx* ctx, int32_t changeover_level, genga_kick_plan* plan)
{
    if (!ctx || !plan) return GENGA_KICK_E_NULL;
    if (changeover_level < 0 || changeover_level > ctx->cfg.max_level) return GENGA_KICK_E_LEVEL;
    *plan = changeover_level == 0 && ctx->plan_sym.n_ctas > 0 ? ctx->plan_sym : ctx->plans[changeover_level];
    return GENGA_KICK_OK;
}

extern "C" int genga_kick_status(genga_kick_ctx* ctx, int32_t* status)
{
    if (!ctx || !status) return GENGA_KICK_E_NULL;
    GK_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    GK_CUDA(ctx, cudaMemcpy(status, ctx->status, sizeof(int), cudaMemcpyDeviceToHost));
    return GENGA_KICK_OK;
}

extern "C" int genga_kick_enable_timing(genga_kick_ctx* ctx, int32_t on)
{
    if (!ctx) return GENGA_KICK_E_NULL;
    const int nl = ctx->cfg.max_level + 1;
    if (on && !ctx->ev) {
        ctx->ev = static_cast<cudaEvent_t*>(std::calloc((size_t)2 * nl, sizeof(cudaEvent_t)));
        ctx->ev_set = static_cast<bool*>(std::calloc((size_t)nl, sizeof(bool)));
        if (!ctx->ev || !ctx->ev_set) return GENGA_KICK_E_NOMEM;
        for (int k = 0; k < 2 * nl; k++) GK_CUDA(ctx, cudaEventCreate(&ctx->ev[k]));
    }
    ctx->timing = on != 0;
    if (ctx->ev_set) std::memset(ctx->ev_set, 0, (size_t)nl * sizeof(bool));
    return GENGA_KICK_OK;
}

extern "C" int genga_kick_last_pair_loop_ms(genga_kick_ctx* ctx, int32_t changeover_level, float* ms)
{
    if (!ctx || !ms) return GENGA_KICK_E_NULL;
    if (changeover_level < 0 || changeover_level > ctx->cfg.max_level) return GENGA_KICK_E_LEVEL;
    if (!ctx->timing || !ctx->ev_set[changeover_level]) return GENGA_KICK_E_SIZE;
    GK_CUDA(ctx, cudaEventSynchronize(ctx->ev[2 * changeover_level + 1]));
    GK_CUDA(ctx, cudaEventElapsedTime(ms, ctx->ev[2 * changeover_level], ctx->ev[2 * changeover_level + 1]));
    return GENGA_KICK_OK;
}

extern "C" int64_t genga_kick_launch_count(const genga_kick_ctx* ctx) { return ctx ? ctx->launches : 0; }

extern "C" int genga_kick_free(genga_kick_ctx* ctx)
{
    if (!ctx) return GENGA_KICK_OK;
    void* bufs[] = {ctx->rxy, ctx->rzm, ctx->rfw, ctx->rfw_ref, ctx->need_near, ctx->ridx, ctx->partial_sym, ctx->react, ctx->sym_t0, ctx->cblo, ctx->cbhi, ctx->bbox, ctx->keys_a,
                    ctx->keys_b, ctx->vals_a, ctx->vals_b, ctx->counts, ctx->partial, ctx->partial2, ctx->status, ctx->cand, ctx->ncand, ctx->fx, ctx->touched, ctx->h_pos,
                    ctx->h_vel, ctx->h_mass, ctx->h_rcrit, ctx->h_acc, ctx->h_pairs, ctx->h_npairs,
                    ctx->psum_partial, ctx->psum_ticket, ctx->step_rcrit, ctx->grp_label, ctx->grp_flag,
                    ctx->grp_keys_a, ctx->grp_keys_b, ctx->grp_vals_a, ctx->grp_vals_b, ctx->grp_counts, ctx->hyb_state, ctx->bs_scratch, ctx->bs_nbr, ctx->senc_slab};
    for (void* b : bufs)
        if (b) cudaFree(b);
    if (ctx->ev)
        for (int k = 0; k < 2 * (ctx->cfg.max_level + 1); k++)
            if (ctx->ev[k]) cudaEventDestroy(ctx->ev[k]);
    std::free(ctx->ev);
    std::free(ctx->ev_set);
    std::free(ctx->plans);
    delete ctx;
    return GENGA_KICK_OK;
}

extern "C" const char* genga_kick_last_cuda_error(const genga_kick_ctx* ctx)
{
    return ctx ? ctx->cuda_err.c_str() : "";
}

// ---------------------------------------------------------------------------------------------------------------------
// genga_kick_list_static (include/genga_kick_static.h): the list kick without a context and without any allocation.
// Its scratch -- the fixed-point accumulators fx[3][GENGA_FX_LIMBS][stride] and the flags touched[N] behind them -- is
// this file-scope array: every device that loads the library holds it until the process exits.  In HOST code the
// array's name is a host-side stand-in, not a device address: static_scratch_of() asks the runtime for the address
// (cudaGetSymbolAddress, once per device, with that device current) and the kernels get that pointer.
// ---------------------------------------------------------------------------------------------------------------------
#include "../../include/genga_kick_static.h"
#include <mutex>

static_assert(GENGA_KICK_STATIC_SCRATCH_BYTES == GENGA_KICK_STATIC_MAX_BODIES * (3 * GENGA_FX_LIMBS * 8 + 4),
              "include/genga_kick_static.h states the size of the accumulators");
static __device__ __align__(256) unsigned long long genga_static_scratch[GENGA_KICK_STATIC_SCRATCH_BYTES / 8];

namespace {

constexpr int kStaticMaxDevices = 64;
struct StaticDevice {
    unsigned long long* scratch;   // device address of genga_static_scratch on this device; nullptr: not asked yet
    int num_sms;
};
StaticDevice g_static_dev[kStaticMaxDevices];
std::mutex g_static_mutex;

// set-up of the current device, once: no allocation (attribute queries and the symbol's address)
int static_scratch_of(StaticDevice& out)
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kStaticMaxDevices) return GENGA_KICK_E_CUDA;
    std::lock_guard<std::mutex> lock(g_static_mutex);
    StaticDevice& d = g_static_dev[dev];
    if (!d.scratch) {
        int major = 0, sms = 0;
        if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) return GENGA_KICK_E_CUDA;
        if (major != 10) return GENGA_KICK_E_CUDA;                                   // sm_100a only
        if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0) return GENGA_KICK_E_CUDA;
        unsigned long long* ptr = nullptr;
        if (cudaGetSymbolAddress(reinterpret_cast<void**>(&ptr), genga_static_scratch) != cudaSuccess || !ptr)
            return GENGA_KICK_E_CUDA;
        d.num_sms = sms;
        d.scratch = ptr;
    }
    out = d;
    return GENGA_KICK_OK;
}

}  // namespace

extern "C" int genga_kick_list_static(const double* pos, double* vel, const double* mass, const double* rcrit,
                                      int64_t n_massive, int64_t n_test, int32_t changeover_level, int32_t tp_mode,
                                      double G, double enc_factor, double dt, const int32_t* in_pairs,
                                      const int32_t* in_n_pairs, int64_t in_pair_rows, double* out_acc, int32_t* out_pairs,
                                      int64_t pair_capacity, int32_t* out_npairs, int32_t* status, void* cuda_stream)
{
    if (!pos || !mass || !rcrit || !in_n_pairs || !out_npairs || !status) return GENGA_KICK_E_NULL;
    if (!out_acc && !vel) return GENGA_KICK_E_NULL;
    if (n_massive < 0 || n_test < 0 || pair_capacity < 0 || in_pair_rows < 0) return GENGA_KICK_E_SIZE;
    if (n_massive > GENGA_MAX_BODIES || n_test > GENGA_MAX_BODIES) return GENGA_KICK_E_SIZE;
    const int64_t N64 = n_massive + n_test;
    if (N64 <= 0 || N64 > GENGA_MAX_BODIES || tp_mode < 0 || tp_mode > 2) return GENGA_KICK_E_SIZE;
    if (N64 > GENGA_KICK_STATIC_MAX_BODIES) return GENGA_KICK_E_STATIC_MAX;
    if (!out_pairs && pair_capacity > 0) return GENGA_KICK_E_NULL;
    if (!in_pairs && in_pair_rows > 0) return GENGA_KICK_E_NULL;
    if (changeover_level < 0 || changeover_level > 62) return GENGA_KICK_E_LEVEL;
    if (misaligned(pos) || misaligned(vel) || misaligned(mass) || misaligned(rcrit) || misaligned(out_acc) ||
        misaligned(out_pairs) || misaligned(out_npairs) || misaligned(in_pairs))
        return GENGA_KICK_E_ALIGN;
    StaticDevice sd = {};
    int rc = static_scratch_of(sd);
    if (rc != GENGA_KICK_OK) return rc;

    const int N = (int)N64;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const long long stride = ((long long)N + 31) / 32 * 32;            // rows of the accumulators: 256-byte multiples
    unsigned long long* fx = sd.scratch;
    int* touched = reinterpret_cast<int*>(sd.scratch + 3 * GENGA_FX_LIMBS * stride);
    // the array keeps what the last call (perhaps one that failed half way) left: clear what this one uses
    const size_t used = (size_t)(3 * GENGA_FX_LIMBS * stride) * sizeof(unsigned long long) + (size_t)N * sizeof(int);
    if (cudaMemsetAsync(sd.scratch, 0, used, st) != cudaSuccess) return GENGA_KICK_E_CUDA;
    if (cudaMemsetAsync(status, 0, sizeof(int32_t), st) != cudaSuccess) return GENGA_KICK_E_CUDA;
    if (cudaMemsetAsync(out_npairs, 0, ((size_t)N + 1) * sizeof(int32_t), st) != cudaSuccess) return GENGA_KICK_E_CUDA;

    genga::KickParams kp = {};
    kp.rcrit = rcrit;
    kp.N = N; kp.n_massive = (int)n_massive; kp.L = changeover_level; kp.f = enc_factor;
    kp.out_pairs = out_pairs; kp.capacity = pair_capacity; kp.out_npairs = out_npairs;
    kp.status = status;
    kp.fx = fx; kp.fx_stride = stride; kp.touched = touched;
    const int blocks = (int)std::min<int64_t>(std::max<int64_t>((in_pair_rows + 1023) / 1024, 1), 8 * sd.num_sms);
    genga::list_kick_kernel<<<blocks, 256, 0, st>>>(kp, pos, mass, G, reinterpret_cast<const int2*>(in_pairs), in_n_pairs,
                                                    in_pair_rows, tp_mode == 2 ? 1 : 0);
    genga::list_reduce_kernel<<<(N + 255) / 256, 256, 0, st>>>(fx, stride, touched, N, dt, status, out_acc, vel);
    return cudaGetLastError() == cudaSuccess ? GENGA_KICK_OK : GENGA_KICK_E_CUDA;
}
