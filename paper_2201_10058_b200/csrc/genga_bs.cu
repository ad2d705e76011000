// C ABI of the Bulirsch-Stoer integration of close-encounter groups (include/genga_bs.h).  Host side only.
#include "../../include/genga_bs.h"
#include "../../include/genga_group.h"
#include "../../include/genga_step.h"
#include "../../include/genga_senc.h"
#include "genga_kick_ctx.h"
#include "genga_bs_kernels.cuh"

#include <algorithm>

extern "C" int genga_bs(genga_kick_ctx* ctx, const double* pos_in, const double* vel_in, const double* mass,
                        const double* rcrit, int32_t nlevels, double m_star, double dt, double tol, const int32_t* members,
                        const int32_t* offsets, const int32_t* summary, double* pos, double* vel)
{
    if (!ctx || !pos_in || !vel_in || !mass || !rcrit || !members || !offsets || !summary || !pos || !vel)
        return GENGA_KICK_E_NULL;
    if (genga_misaligned(pos_in) || genga_misaligned(vel_in) || genga_misaligned(mass) || genga_misaligned(rcrit) ||
        genga_misaligned(members) || genga_misaligned(offsets) || genga_misaligned(summary) || genga_misaligned(pos) ||
        genga_misaligned(vel))
        return GENGA_KICK_E_ALIGN;
    if (nlevels < 1 || nlevels > GENGA_BS_MAX_LEVELS || !(m_star > 0.0) || !(tol > 0.0) || pos == pos_in || vel == vel_in)
        return GENGA_KICK_E_SIZE;
    if (dt == 0.0) return GENGA_KICK_OK;
    const long long N = ctx->N;
    cudaStream_t st = ctx->stream;
    const double G = ctx->cfg.G, mu = ctx->cfg.G * m_star;
    int* status = ctx->status;
    long long NN = N;
    // test-particle modes (sec. 8.1): bodies from n_massive on are semi-active particles; TP 0 has none
    long long n_massive = ctx->cfg.n_test > 0 ? (long long)ctx->cfg.n_massive : N;
    int tp_mode = ctx->cfg.tp_mode;
    // whole-grid regime: scratch for one group of up to N bodies, and the size of a co-resident grid
    if (!ctx->bs_scratch) {
        const size_t bytes = ((size_t)(7 + GENGA_BS_MAX_LEVELS) * N + 8) * sizeof(double);
        GK_CUDA(ctx, cudaMalloc(&ctx->bs_scratch, bytes));
        GK_CUDA(ctx, cudaMemsetAsync(ctx->bs_scratch, 0, bytes, st));
        int per_sm = 0;
        GK_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, genga::bs_kernel<GENGA_BS_MODE_COOP, GENGA_BS_COOP_THREADS, GENGA_BS_SUB>,
                                                                 GENGA_BS_COOP_THREADS, 0));
        if (per_sm < 1) return genga_cuda_fail(ctx, cudaErrorLaunchOutOfResources);
        ctx->bs_coop_blocks = per_sm * ctx->num_sms;
        GK_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(
                         &per_sm, genga::bs_kernel<GENGA_BS_MODE_COOP, GENGA_BS_COOP_THREADS, 1>, GENGA_BS_COOP_THREADS, 0));
        if (per_sm < 1) return genga_cuda_fail(ctx, cudaErrorLaunchOutOfResources);
        ctx->bs_coop_blocks1 = per_sm * ctx->num_sms;
    }
    genga::BsGlobal gm;
    {
        double* p = ctx->bs_scratch;
        for (int h = 0; h < 2; h++) { gm.x[h] = p; p += N; gm.y[h] = p; p += N; gm.z[h] = p; p += N; }
        gm.gm = p; p += N;
        for (int k = 0; k < GENGA_BS_MAX_LEVELS; k++) { gm.rc[k] = p; p += N; }
        gm.err = reinterpret_cast<unsigned long long*>(p);
        gm.totals = gm.err + 4;
        gm.stats = reinterpret_cast<int4*>(ctx->bs_stats);
        gm.stats_rows = ctx->bs_stats_rows;
    }
    // at most N / 2 groups; warps / CTAs stride over them (their number is only known on the device)
    int small_max = GENGA_BS_THREADS;
    // one launch: one warp per group of up to 8 bodies (nearly all groups), eight groups per CTA, in the first `wblocks`
    // CTAs; one CTA per group of 9 .. 32 bodies, eight lanes per body, in the rest
    {
        const int wblocks = (int)std::min<long long>(std::max<long long>((N / 2 + 7) / 8, 1), 8LL * ctx->num_sms);
        const int cblocks = N > GENGA_BS_SEQ_MAX
                                ? (int)std::min<long long>(std::max<long long>(N / (GENGA_BS_SEQ_MAX + 1), 1), 4LL * ctx->num_sms)
                                : 0;
        genga::bs_small_kernel<<<wblocks + cblocks, GENGA_BS_THREADS, 0, st>>>(
            pos_in, vel_in, mass, rcrit, NN, nlevels, G, mu, dt, tol, members, offsets, summary, pos, vel, status, gm, small_max,
            n_massive, tp_mode, -1, wblocks);
    }
    // one cluster of 8 CTAs per group of 33 .. 256 bodies, eight lanes per body
    if (N > GENGA_BS_WARP_MAX) {
        const long long clusters = std::min<long long>(std::max<long long>(N / (GENGA_BS_WARP_MAX + 1), 1),
                                                       2LL * ctx->num_sms / GENGA_BS_CLUSTER);
        int lo = GENGA_BS_WARP_MAX;
        genga::bs_cluster_kernel<<<(unsigned)(clusters * GENGA_BS_CLUSTER), GENGA_BS_THREADS, 0, st>>>(
            pos_in, vel_in, mass, rcrit, NN, nlevels, G, mu, dt, tol, members, offsets, summary, pos, vel, status, gm, lo,
            n_massive, tp_mode, -1);
        ctx->launches++;
    }
    GK_CUDA(ctx, cudaGetLastError());
    // the whole-grid regime, one large group after the other (returns at once if there is none): first a grid of one
    // CTA per SM for the groups it can hold (its grid barrier costs a fraction of the full grid's), then the full
    // co-resident grid for the larger ones
    if (N > GENGA_BS_THREADS) {
        GK_CUDA(ctx, cudaMemsetAsync(gm.err, 0, 4 * sizeof(unsigned long long), st));
        const int cap1 = ctx->num_sms * GENGA_BS_COOP_THREADS / GENGA_BS_SUB;
        const bool two = N > cap1 && ctx->bs_coop_blocks > ctx->num_sms;
        int big_max = two ? cap1 : -1;
        void* args[] = {&pos_in, &vel_in, &mass, &rcrit, &NN, &nlevels, const_cast<double*>(&G), const_cast<double*>(&mu), &dt,
                        &tol, &members, &offsets, &summary, &pos, &vel, &status, &gm, &small_max, &n_massive, &tp_mode, &big_max};
        GK_CUDA(ctx, cudaLaunchCooperativeKernel(reinterpret_cast<void*>(genga::bs_kernel<GENGA_BS_MODE_COOP, GENGA_BS_COOP_THREADS, GENGA_BS_SUB>),
                                                 dim3(two ? ctx->num_sms : ctx->bs_coop_blocks), dim3(GENGA_BS_COOP_THREADS), args, 0,
                                                 st));
        ctx->launches++;
        if (two) {
            // ... the full grid with eight lanes per body, and with one lane per body for the groups beyond that
            const int cap2 = (int)std::min<long long>((long long)ctx->bs_coop_blocks * GENGA_BS_COOP_THREADS / GENGA_BS_SUB, N);
            const bool three = N > cap2;
            small_max = cap1;
            big_max = three ? cap2 : -1;
            GK_CUDA(ctx, cudaMemsetAsync(gm.err, 0, 4 * sizeof(unsigned long long), st));
            GK_CUDA(ctx, cudaLaunchCooperativeKernel(reinterpret_cast<void*>(genga::bs_kernel<GENGA_BS_MODE_COOP, GENGA_BS_COOP_THREADS, GENGA_BS_SUB>),
                                                     dim3(ctx->bs_coop_blocks), dim3(GENGA_BS_COOP_THREADS), args, 0, st));
            ctx->launches++;
            if (three) {
                small_max = cap2;
                big_max = -1;
                GK_CUDA(ctx, cudaMemsetAsync(gm.err, 0, 4 * sizeof(unsigned long long), st));
                GK_CUDA(ctx, cudaLaunchCooperativeKernel(
                                 reinterpret_cast<void*>(genga::bs_kernel<GENGA_BS_MODE_COOP, GENGA_BS_COOP_THREADS, 1>),
                                 dim3(ctx->bs_coop_blocks1), dim3(GENGA_BS_COOP_THREADS), args, 0, st));
                ctx->launches++;
            }
        }
    }
    GK_CUDA(ctx, cudaGetLastError());
    ctx->launches++;
    return GENGA_KICK_OK;
}

extern "C" int genga_bs_set_stats(genga_kick_ctx* ctx, int32_t* group_stats, int64_t rows)
{
    if (!ctx) return GENGA_KICK_E_NULL;
    if (rows < 0 || (rows > 0 && !group_stats)) return GENGA_KICK_E_SIZE;
    if (genga_misaligned(group_stats)) return GENGA_KICK_E_ALIGN;
    ctx->bs_stats = group_stats;
    ctx->bs_stats_rows = group_stats ? rows : 0;
    return GENGA_KICK_OK;
}

extern "C" int genga_bs_totals(genga_kick_ctx* ctx, int64_t* totals, int32_t reset)
{
    if (!ctx || !totals) return GENGA_KICK_E_NULL;
    totals[0] = totals[1] = totals[2] = totals[3] = 0;
    if (!ctx->bs_scratch) return GENGA_KICK_OK;                       // genga_bs has not run yet
    unsigned long long* t = reinterpret_cast<unsigned long long*>(ctx->bs_scratch + (size_t)(7 + GENGA_BS_MAX_LEVELS) * ctx->N) + 4;
    GK_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    GK_CUDA(ctx, cudaMemcpy(totals, t, 4 * sizeof(int64_t), cudaMemcpyDeviceToHost));
    if (reset) GK_CUDA(ctx, cudaMemset(t, 0, 4 * sizeof(int64_t)));
    return GENGA_KICK_OK;
}

extern "C" int genga_hybrid_step(genga_kick_ctx* ctx, double* pos, double* vel, const double* mass, double m_star, double dt,
                                 double n1, double n2, double tol, double* out_acc, int32_t* out_pairs, int32_t* out_npairs,
                                 int32_t* group_of, int32_t* members, int32_t* offsets, int32_t* summary)
{
    if (!ctx || !pos || !vel || !mass || !out_npairs || !group_of || !members || !offsets || !summary)
        return GENGA_KICK_E_NULL;
    if (!out_pairs && ctx->cfg.pair_capacity > 0) return GENGA_KICK_E_NULL;
    const size_t N = (size_t)ctx->N;
    if (!ctx->step_rcrit) GK_CUDA(ctx, cudaMalloc(&ctx->step_rcrit, N * sizeof(double)));
    if (!ctx->hyb_state) GK_CUDA(ctx, cudaMalloc(&ctx->hyb_state, 6 * N * sizeof(double)));
    double* q_in = ctx->hyb_state;
    double* v_in = ctx->hyb_state + 3 * N;
    cudaStream_t st = ctx->stream;
    int rc = genga_rcrit(ctx, pos, vel, mass, m_star, dt, 2.0, 1, n1, n2, ctx->step_rcrit);
    if (rc != GENGA_KICK_OK) return rc;
    rc = genga_kick(ctx, pos, vel, mass, ctx->step_rcrit, 0, 0.5 * dt, nullptr, out_pairs, out_npairs);
    if (rc != GENGA_KICK_OK) return rc;
    rc = genga_hc(ctx, pos, vel, mass, m_star, 0.5 * dt);
    if (rc != GENGA_KICK_OK) return rc;
    GK_CUDA(ctx, cudaMemcpyAsync(q_in, pos, 3 * N * sizeof(double), cudaMemcpyDeviceToDevice, st));
    GK_CUDA(ctx, cudaMemcpyAsync(v_in, vel, 3 * N * sizeof(double), cudaMemcpyDeviceToDevice, st));
    rc = genga_fg(ctx, pos, vel, m_star, dt);
    if (rc != GENGA_KICK_OK) return rc;
    rc = genga_group_impl(ctx, out_pairs, out_npairs + N, ctx->cfg.pair_capacity, group_of, members, offsets, summary,
                          GENGA_KICK_STATUS_LIST_CLIPPED);
    if (rc != GENGA_KICK_OK) return rc;
    rc = genga_bs(ctx, q_in, v_in, mass, ctx->step_rcrit, 1, m_star, dt, tol, members, offsets, summary, pos, vel);
    if (rc != GENGA_KICK_OK) return rc;
    rc = genga_hc(ctx, pos, vel, mass, m_star, 0.5 * dt);
    if (rc != GENGA_KICK_OK) return rc;
    return genga_kick_impl(ctx, pos, vel, mass, ctx->step_rcrit, 0, 0.5 * dt, out_acc, nullptr, nullptr);
}
