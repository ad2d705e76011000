// C ABI of the Bulirsch-Stoer integration of close-encounter groups (include/genga_bs.h).  Host side only.
#include "../../include/genga_bs.h"
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
    // at most N / 2 groups; CTAs stride over them (the number of groups is only known on the device)
    const int blocks = (int)std::min<long long>(std::max<long long>(N / 2, 1), 16LL * ctx->num_sms);
    genga::bs_kernel<<<blocks, GENGA_BS_THREADS, 0, ctx->stream>>>(pos_in, vel_in, mass, rcrit, N, nlevels, ctx->cfg.G,
                                                                  ctx->cfg.G * m_star, dt, tol, members, offsets, summary,
                                                                  pos, vel, ctx->status);
    GK_CUDA(ctx, cudaGetLastError());
    ctx->launches++;
    return GENGA_KICK_OK;
}
