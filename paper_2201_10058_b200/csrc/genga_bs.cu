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
    // whole-grid regime: the size of a co-resident grid, and scratch for one group of up to N bodies or for one group
    // of up to GENGA_BS_TEAM_BODIES bodies per team
    if (!ctx->bs_scratch) {
        int per_sm = 0;
        GK_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, genga::bs_kernel<GENGA_BS_MODE_COOP, GENGA_BS_COOP_THREADS, GENGA_BS_SUB>,
                                                                 GENGA_BS_COOP_THREADS, 0));
        if (per_sm < 1) return genga_cuda_fail(ctx, cudaErrorLaunchOutOfResources);
        ctx->bs_coop_blocks = per_sm * ctx->num_sms;
        GK_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(
                         &per_sm, genga::bs_kernel<GENGA_BS_MODE_COOP, GENGA_BS_COOP_THREADS, 1>, GENGA_BS_COOP_THREADS, 0));
        if (per_sm < 1) return genga_cuda_fail(ctx, cudaErrorLaunchOutOfResources);
        ctx->bs_coop_blocks1 = per_sm * ctx->num_sms;
        ctx->bs_coop_blocks_by_lanes[0] = ctx->bs_coop_blocks;
        ctx->bs_coop_blocks_by_lanes[3] = ctx->bs_coop_blocks1;
        GK_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(
                         &per_sm, genga::bs_kernel<GENGA_BS_MODE_COOP, GENGA_BS_COOP_THREADS, 4>, GENGA_BS_COOP_THREADS, 0));
        if (per_sm < 1) return genga_cuda_fail(ctx, cudaErrorLaunchOutOfResources);
        ctx->bs_coop_blocks_by_lanes[1] = per_sm * ctx->num_sms;
        GK_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(
                         &per_sm, genga::bs_kernel<GENGA_BS_MODE_COOP, GENGA_BS_COOP_THREADS, 2>, GENGA_BS_COOP_THREADS, 0));
        if (per_sm < 1) return genga_cuda_fail(ctx, cudaErrorLaunchOutOfResources);
        ctx->bs_coop_blocks_by_lanes[2] = per_sm * ctx->num_sms;
        ctx->bs_teams = ctx->bs_coop_blocks / GENGA_BS_TEAM_CTAS;           // most teams any launch forms
        ctx->bs_rows = std::max<long long>(N, (long long)ctx->bs_coop_blocks * GENGA_BS_COOP_THREADS / GENGA_BS_SUB);
        for (int v = 1, lanes = GENGA_BS_SUB / 2; v < 4; v++, lanes /= 2)
            ctx->bs_rows = std::max<long long>(ctx->bs_rows, lanes > 1 ? (long long)ctx->bs_coop_blocks_by_lanes[v] * GENGA_BS_COOP_THREADS / lanes : N);
        const size_t bytes = ((size_t)(28 + GENGA_BS_MAX_LEVELS) * ctx->bs_rows + 16 * (size_t)std::max(ctx->bs_teams, 1) + 8) * sizeof(double);
        GK_CUDA(ctx, cudaMalloc(&ctx->bs_scratch, bytes));
        GK_CUDA(ctx, cudaMemsetAsync(ctx->bs_scratch, 0, bytes, st));
        if (N > GENGA_BS_THREADS) {
            // neighbour lists of the whole-grid regime: room for 1024 partners per body of the context (at least 2^24
            // entries, at most 2^28), shared out among the teams; a group whose lists need more falls back to all pairs
            ctx->bs_nbr_capacity = std::min<long long>(std::max<long long>(1024LL * N, 1LL << 24), 1LL << 28);
            GK_CUDA(ctx, cudaMalloc(&ctx->bs_nbr, (size_t)ctx->bs_nbr_capacity * sizeof(int)));
        }
    }
    genga::BsGlobal gm = {};
    const size_t ctrl_words = 16 * (size_t)std::max(ctx->bs_teams, 1);
    {
        const long long R = ctx->bs_rows;
        double* p = ctx->bs_scratch;
        for (int h = 0; h < 2; h++) { gm.pk[h] = reinterpret_cast<double2*>(p); p += 4 * R; }     // (16-byte aligned: first)
        gm.sr = reinterpret_cast<double2*>(p); p += 6 * R;
        for (int h = 0; h < 2; h++) { gm.x[h] = p; p += R; gm.y[h] = p; p += R; gm.z[h] = p; p += R; }
        gm.gm = p; p += R;
        gm.rcsq = p; p += R;
        gm.lr = p; p += R;
        gm.la = p; p += R;
        gm.ld = p; p += R;
        gm.vx = p; p += R; gm.vy = p; p += R; gm.vz = p; p += R;
        for (int k = 0; k < GENGA_BS_MAX_LEVELS; k++) { gm.rc[k] = p; p += R; }
        gm.err = reinterpret_cast<unsigned long long*>(p);               // [teams][16] control words, then totals[4]
        gm.totals = gm.err + ctrl_words;
        gm.nbr = ctx->bs_nbr;
        gm.nbr_capacity = ctx->bs_nbr_capacity;
        gm.stats = reinterpret_cast<int4*>(ctx->bs_stats);
        gm.stats_rows = ctx->bs_stats_rows;
        gm.team_ctas = 0;
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
    // groups above 256 bodies: cooperative launches (co-resident CTAs), eight lanes per body.  First the groups of up
    // to 512 and then of up to 2048 bodies, several at a time: the grid cut into teams of 64 resp. 256 CTAs, a team per
    // group with a barrier of its own.  Then the larger ones, one after the other over the whole grid, while the grid
    // holds them at eight lanes per body (~11,800 bodies); one lane per body beyond.  Every launch returns at once if
    // summary[2] shows no group for it.
    if (N > GENGA_BS_THREADS) {
        int big_max = 0;
        void* args[] = {&pos_in, &vel_in, &mass, &rcrit, &NN, &nlevels, const_cast<double*>(&G), const_cast<double*>(&mu), &dt,
                        &tol, &members, &offsets, &summary, &pos, &vel, &status, &gm, &small_max, &n_massive, &tp_mode, &big_max};
        void* k8 = reinterpret_cast<void*>(genga::bs_kernel<GENGA_BS_MODE_COOP, GENGA_BS_COOP_THREADS, GENGA_BS_SUB>);
        void* k1 = reinterpret_cast<void*>(genga::bs_kernel<GENGA_BS_MODE_COOP, GENGA_BS_COOP_THREADS, 1>);
        small_max = GENGA_BS_THREADS;
        for (int mult = 1; mult <= 4; mult *= 4) {                          // teams of 16 and of 64 CTAs (4096 and 16,384 lanes)
            const int tctas = GENGA_BS_TEAM_CTAS * mult, teams = ctx->bs_coop_blocks / tctas;
            const int cap = tctas * GENGA_BS_COOP_THREADS / GENGA_BS_SUB;
            if (teams < 2 || N <= small_max) continue;
            big_max = N > cap ? cap : -1;
            gm.team_ctas = tctas;
            GK_CUDA(ctx, cudaMemsetAsync(gm.err, 0, ctrl_words * sizeof(unsigned long long), st));
            GK_CUDA(ctx, cudaLaunchCooperativeKernel(k8, dim3(teams * tctas), dim3(GENGA_BS_COOP_THREADS), args, 0, st));
            ctx->launches++;
            small_max = cap;
        }
        gm.team_ctas = 0;
        // the whole grid on one group at a time: as many lanes per body as the grid has for the group's size
        void* kern[4] = {k8,
                         reinterpret_cast<void*>(genga::bs_kernel<GENGA_BS_MODE_COOP, GENGA_BS_COOP_THREADS, 4>),
                         reinterpret_cast<void*>(genga::bs_kernel<GENGA_BS_MODE_COOP, GENGA_BS_COOP_THREADS, 2>), k1};
        for (int v = 0, lanes = GENGA_BS_SUB; v < 4 && N > small_max; v++, lanes /= 2) {
            const long long cap = lanes > 1 ? (long long)ctx->bs_coop_blocks_by_lanes[v] * GENGA_BS_COOP_THREADS / lanes : N;
            if (cap <= small_max) continue;
            big_max = N > cap ? (int)cap : -1;
            GK_CUDA(ctx, cudaMemsetAsync(gm.err, 0, ctrl_words * sizeof(unsigned long long), st));
            GK_CUDA(ctx, cudaLaunchCooperativeKernel(kern[v], dim3(ctx->bs_coop_blocks_by_lanes[v]), dim3(GENGA_BS_COOP_THREADS),
                                                     args, 0, st));
            ctx->launches++;
            small_max = (int)std::min<long long>(cap, N);
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
    unsigned long long* t = reinterpret_cast<unsigned long long*>(ctx->bs_scratch + (size_t)(28 + GENGA_BS_MAX_LEVELS) * ctx->bs_rows) +
                            16 * (size_t)std::max(ctx->bs_teams, 1);
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
