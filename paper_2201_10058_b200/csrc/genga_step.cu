// C ABI of the O(N) neighbours of the kick and of the composed step (include/genga_step.h).
// Host side only: argument checks, scratch, kernel launches on the context's stream.
#include "../../include/genga_step.h"
#include "genga_kick_ctx.h"
#include "genga_step_kernels.cuh"

#include <algorithm>

namespace {

int ensure_step_scratch(genga_kick_ctx* ctx)
{
    if (!ctx->psum_partial) {
        // rows [0, GENGA_PSUM_BLOCKS): CTA partial sums; rows GENGA_PSUM_BLOCKS + {0, 1}: totals
        GK_CUDA(ctx, cudaMalloc(&ctx->psum_partial, (size_t)3 * (GENGA_PSUM_BLOCKS + 2) * sizeof(double)));
    }
    if (!ctx->psum_ticket) {
        GK_CUDA(ctx, cudaMalloc(&ctx->psum_ticket, 16));
        GK_CUDA(ctx, cudaMemsetAsync(ctx->psum_ticket, 0, 16, ctx->stream));
    }
    return GENGA_KICK_OK;
}

}  // namespace

extern "C" int genga_rcrit(genga_kick_ctx* ctx, const double* pos, const double* vel, const double* mass, double m_star,
                           double dt, double substeps, int32_t nrows, double n1, double n2, double* out_rcrit)
{
    if (!ctx || !pos || !vel || !mass || !out_rcrit) return GENGA_KICK_E_NULL;
    if (genga_misaligned(pos) || genga_misaligned(vel) || genga_misaligned(mass) || genga_misaligned(out_rcrit))
        return GENGA_KICK_E_ALIGN;
    if (nrows < 1 || !(substeps > 0.0) || !(m_star > 0.0)) return GENGA_KICK_E_SIZE;
    const long long N = ctx->N;
    genga::rcrit_kernel<<<genga::step_blocks(N), GENGA_STEP_THREADS, 0, ctx->stream>>>(
        pos, vel, mass, N, ctx->cfg.G * m_star, m_star, dt, substeps, nrows, n1, n2, out_rcrit, ctx->status, nullptr,
        nullptr, 0);
    GK_CUDA(ctx, cudaGetLastError());
    ctx->launches++;
    return GENGA_KICK_OK;
}

extern "C" int genga_rcrit_list(genga_kick_ctx* ctx, const double* pos, const double* vel, const double* mass,
                                double m_star, double dt, double substeps, int32_t nrows, double n1, double n2,
                                const int32_t* list, const int32_t* n_list, int64_t list_rows, double* out_rcrit)
{
    if (!ctx || !pos || !vel || !mass || !out_rcrit || !list || !n_list) return GENGA_KICK_E_NULL;
    if (genga_misaligned(pos) || genga_misaligned(vel) || genga_misaligned(mass) || genga_misaligned(out_rcrit) ||
        genga_misaligned(list))
        return GENGA_KICK_E_ALIGN;
    if (nrows < 1 || !(substeps > 0.0) || !(m_star > 0.0) || list_rows < 0) return GENGA_KICK_E_SIZE;
    const long long N = ctx->N;
    const int blocks = (int)std::min<long long>(std::max<long long>((list_rows + GENGA_STEP_THREADS - 1) / GENGA_STEP_THREADS, 1),
                                                GENGA_PSUM_BLOCKS);
    genga::rcrit_kernel<<<blocks, GENGA_STEP_THREADS, 0, ctx->stream>>>(
        pos, vel, mass, N, ctx->cfg.G * m_star, m_star, dt, substeps, nrows, n1, n2, out_rcrit, ctx->status, list, n_list,
        list_rows);
    GK_CUDA(ctx, cudaGetLastError());
    ctx->launches++;
    return GENGA_KICK_OK;
}

extern "C" int genga_fg_list(genga_kick_ctx* ctx, double* pos, double* vel, double m_star, double dt, const int32_t* list,
                             const int32_t* n_list, int64_t list_rows)
{
    if (!ctx || !pos || !vel || !list || !n_list) return GENGA_KICK_E_NULL;
    if (genga_misaligned(pos) || genga_misaligned(vel) || genga_misaligned(list)) return GENGA_KICK_E_ALIGN;
    if (!(m_star > 0.0) || list_rows < 0) return GENGA_KICK_E_SIZE;
    const int blocks = (int)std::min<long long>(std::max<long long>((list_rows + GENGA_STEP_THREADS - 1) / GENGA_STEP_THREADS, 1),
                                                GENGA_PSUM_BLOCKS);
    genga::fg_list_kernel<<<blocks, GENGA_STEP_THREADS, 0, ctx->stream>>>(pos, vel, ctx->N, ctx->cfg.G * m_star, dt, list,
                                                                         n_list, list_rows, ctx->status);
    GK_CUDA(ctx, cudaGetLastError());
    ctx->launches++;
    return GENGA_KICK_OK;
}

extern "C" int genga_hc(genga_kick_ctx* ctx, double* pos, const double* vel, const double* mass, double m_star, double dt)
{
    if (!ctx || !pos || !vel || !mass) return GENGA_KICK_E_NULL;
    if (genga_misaligned(pos) || genga_misaligned(vel) || genga_misaligned(mass)) return GENGA_KICK_E_ALIGN;
    if (!(m_star > 0.0)) return GENGA_KICK_E_SIZE;
    int rc = ensure_step_scratch(ctx);
    if (rc != GENGA_KICK_OK) return rc;
    const long long N = ctx->N;
    const int nb = genga::step_blocks(N);
    genga::psum_kernel<<<nb, GENGA_STEP_THREADS, 0, ctx->stream>>>(vel, mass, N, ctx->psum_partial, ctx->psum_ticket, 0);
    genga::shift_kernel<<<nb, GENGA_STEP_THREADS, 0, ctx->stream>>>(pos, N, ctx->psum_partial, 0, dt, m_star);
    GK_CUDA(ctx, cudaGetLastError());
    ctx->launches += 2;
    return GENGA_KICK_OK;
}

extern "C" int genga_fg(genga_kick_ctx* ctx, double* pos, double* vel, double m_star, double dt)
{
    if (!ctx || !pos || !vel) return GENGA_KICK_E_NULL;
    if (genga_misaligned(pos) || genga_misaligned(vel)) return GENGA_KICK_E_ALIGN;
    if (!(m_star > 0.0)) return GENGA_KICK_E_SIZE;
    const long long N = ctx->N;
    genga::fg_kernel<false><<<genga::step_blocks(N), GENGA_STEP_THREADS, 0, ctx->stream>>>(
        pos, vel, nullptr, N, ctx->cfg.G * m_star, dt, 0.0, m_star, nullptr, nullptr, 0, 0, ctx->status);
    GK_CUDA(ctx, cudaGetLastError());
    ctx->launches++;
    return GENGA_KICK_OK;
}

extern "C" int genga_drift(genga_kick_ctx* ctx, double* pos, double* vel, const double* mass, double m_star, double dt)
{
    if (!ctx || !pos || !vel || !mass) return GENGA_KICK_E_NULL;
    if (genga_misaligned(pos) || genga_misaligned(vel) || genga_misaligned(mass)) return GENGA_KICK_E_ALIGN;
    if (!(m_star > 0.0)) return GENGA_KICK_E_SIZE;
    int rc = ensure_step_scratch(ctx);
    if (rc != GENGA_KICK_OK) return rc;
    const long long N = ctx->N;
    const int nb = genga::step_blocks(N);
    const double h = 0.5 * dt;
    cudaStream_t st = ctx->stream;
    genga::psum_kernel<<<nb, GENGA_STEP_THREADS, 0, st>>>(vel, mass, N, ctx->psum_partial, ctx->psum_ticket, 0);
    genga::fg_kernel<true><<<nb, GENGA_STEP_THREADS, 0, st>>>(pos, vel, mass, N, ctx->cfg.G * m_star, dt, h, m_star,
                                                              ctx->psum_partial, ctx->psum_ticket, 0, 1, ctx->status);
    genga::shift_kernel<<<nb, GENGA_STEP_THREADS, 0, st>>>(pos, N, ctx->psum_partial, 1, h, m_star);
    GK_CUDA(ctx, cudaGetLastError());
    ctx->launches += 3;
    return GENGA_KICK_OK;
}

extern "C" int genga_step(genga_kick_ctx* ctx, double* pos, double* vel, const double* mass, double m_star, double dt,
                          double n1, double n2, double* rcrit_row, double* out_acc, int32_t* out_pairs,
                          int32_t* out_npairs)
{
    if (!ctx || !pos || !vel || !mass || !out_npairs) return GENGA_KICK_E_NULL;
    if (genga_misaligned(rcrit_row)) return GENGA_KICK_E_ALIGN;
    if (!rcrit_row) {
        if (!ctx->step_rcrit) GK_CUDA(ctx, cudaMalloc(&ctx->step_rcrit, (size_t)ctx->N * sizeof(double)));
        rcrit_row = ctx->step_rcrit;
    }
    int rc = genga_rcrit(ctx, pos, vel, mass, m_star, dt, 2.0, 1, n1, n2, rcrit_row);
    if (rc != GENGA_KICK_OK) return rc;
    rc = genga_kick(ctx, pos, vel, mass, rcrit_row, 0, 0.5 * dt, nullptr, out_pairs, out_npairs);
    if (rc != GENGA_KICK_OK) return rc;
    rc = genga_drift(ctx, pos, vel, mass, m_star, dt);
    if (rc != GENGA_KICK_OK) return rc;
    return genga_kick_impl(ctx, pos, vel, mass, rcrit_row, 0, 0.5 * dt, out_acc, nullptr, nullptr);
}
