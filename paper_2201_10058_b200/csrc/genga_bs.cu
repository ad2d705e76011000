// C ABI of the Bulirsch-Stoer integration of close-encounter groups (include/genga_bs.h).  Host side only.
#include "../../include/genga_bs.h"
#include "../../include/genga_group.h"
#include "../../include/genga_step.h"
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
    static bool configured[64] = {};                          // per device: the kernel needs 64 KB of dynamic shared memory
    const int dev = ctx->cfg.device;
    if (dev >= 0 && dev < 64 && !configured[dev]) {
        GK_CUDA(ctx, cudaFuncSetAttribute(genga::bs_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          (int)genga::bs_smem_bytes()));
        configured[dev] = true;
    }
    genga::bs_kernel<<<blocks, GENGA_BS_THREADS, genga::bs_smem_bytes(), ctx->stream>>>(pos_in, vel_in, mass, rcrit, N, nlevels, ctx->cfg.G,
                                                                  ctx->cfg.G * m_star, dt, tol, members, offsets, summary,
                                                                  pos, vel, ctx->status);
    GK_CUDA(ctx, cudaGetLastError());
    ctx->launches++;
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
    rc = genga_group(ctx, out_pairs, out_npairs + N, ctx->cfg.pair_capacity, group_of, members, offsets, summary);
    if (rc != GENGA_KICK_OK) return rc;
    rc = genga_bs(ctx, q_in, v_in, mass, ctx->step_rcrit, 1, m_star, dt, tol, members, offsets, summary, pos, vel);
    if (rc != GENGA_KICK_OK) return rc;
    rc = genga_hc(ctx, pos, vel, mass, m_star, 0.5 * dt);
    if (rc != GENGA_KICK_OK) return rc;
    return genga_kick_impl(ctx, pos, vel, mass, ctx->step_rcrit, 0, 0.5 * dt, out_acc, nullptr, nullptr);
}
