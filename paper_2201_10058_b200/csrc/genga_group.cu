// C ABI of the grouping of close-encounter pairs (include/genga_group.h).  Host side only.
#include "../../include/genga_group.h"
#include "genga_kick_ctx.h"
#include "genga_kick_sort.cuh"
#include "genga_group_kernels.cuh"

#include <algorithm>

namespace {

const int GENGA_GROUP_SAMPLE = 8;      // first hook pass: every 8th pair

int ensure_group_scratch(genga_kick_ctx* ctx)
{
    if (ctx->grp_label) return GENGA_KICK_OK;
    const size_t N = (size_t)ctx->N;
    const size_t nb = (N + genga::genga_sort_block((long long)N) - 1) / genga::genga_sort_block((long long)N);
    GK_CUDA(ctx, cudaMalloc(&ctx->grp_label, N * sizeof(int)));
    GK_CUDA(ctx, cudaMalloc(&ctx->grp_flag, N * sizeof(int)));
    GK_CUDA(ctx, cudaMalloc(&ctx->grp_keys_a, N * sizeof(unsigned)));
    GK_CUDA(ctx, cudaMalloc(&ctx->grp_keys_b, N * sizeof(unsigned)));
    GK_CUDA(ctx, cudaMalloc(&ctx->grp_vals_a, N * sizeof(int)));
    GK_CUDA(ctx, cudaMalloc(&ctx->grp_vals_b, N * sizeof(int)));
    GK_CUDA(ctx, cudaMalloc(&ctx->grp_counts, (size_t)GENGA_SORT_MAXDIGITS * nb * sizeof(int)));
    return GENGA_KICK_OK;
}

}  // namespace

extern "C" int genga_group(genga_kick_ctx* ctx, const int32_t* pairs, const int32_t* n_pairs, int64_t pair_rows,
                           int32_t* group_of, int32_t* members, int32_t* offsets, int32_t* summary)
{
    return genga_group_impl(ctx, pairs, n_pairs, pair_rows, group_of, members, offsets, summary, 0);
}

int genga_group_impl(genga_kick_ctx* ctx, const int32_t* pairs, const int32_t* n_pairs, int64_t pair_rows,
                     int32_t* group_of, int32_t* members, int32_t* offsets, int32_t* summary, int clip_status)
{
    if (!ctx || !n_pairs || !group_of || !members || !offsets || !summary) return GENGA_KICK_E_NULL;
    if (pair_rows < 0) return GENGA_KICK_E_SIZE;
    if (!pairs && pair_rows > 0) return GENGA_KICK_E_NULL;
    if (genga_misaligned(pairs) || genga_misaligned(group_of) || genga_misaligned(members) || genga_misaligned(offsets) ||
        genga_misaligned(summary))
        return GENGA_KICK_E_ALIGN;
    int rc = ensure_group_scratch(ctx);
    if (rc != GENGA_KICK_OK) return rc;

    const int N = (int)ctx->N;
    const int blocks = (N + 255) / 256;
    cudaStream_t st = ctx->stream;
    genga::group_init_kernel<<<blocks, 256, 0, st>>>(ctx->grp_label, ctx->grp_flag, N, offsets, summary);
    const int hook_blocks = (int)std::min<int64_t>(std::max<int64_t>((pair_rows + 255) / 256, 1), 8 * ctx->num_sms);
    const int2* pr = reinterpret_cast<const int2*>(pairs);
    genga::group_hook_kernel<<<hook_blocks, 256, 0, st>>>(pr, n_pairs, pair_rows, N, GENGA_GROUP_SAMPLE, true, ctx->grp_label,
                                                          ctx->grp_flag, summary, ctx->status, clip_status);
    genga::group_compress_kernel<<<blocks, 256, 0, st>>>(ctx->grp_label, N);
    genga::group_hook_kernel<<<hook_blocks, 256, 0, st>>>(pr, n_pairs, pair_rows, N, GENGA_GROUP_SAMPLE, false, ctx->grp_label,
                                                          ctx->grp_flag, summary, ctx->status, clip_status);
    genga::group_flat_kernel<<<blocks, 256, 0, st>>>(ctx->grp_label, ctx->grp_flag, N, group_of, ctx->grp_keys_a,
                                                     ctx->grp_vals_a);
    ctx->launches += 5;

    // stable LSD radix sort of (key, body) by key in [0, N]: digits of at most 9 bits (GENGA_SORT_MAXDIGITS)
    int key_bits = 1;
    while ((1ll << key_bits) <= (long long)N) key_bits++;
    const int sb = genga::genga_sort_block(N), nb = (N + sb - 1) / sb;
    unsigned *ka = ctx->grp_keys_a, *kb = ctx->grp_keys_b;
    int *va = ctx->grp_vals_a, *vb = ctx->grp_vals_b;
    const int passes = (key_bits + 8) / 9;
    for (int pass = 0, shift = 0; pass < passes; pass++) {
        const int bits = (key_bits - shift + (passes - pass) - 1) / (passes - pass);      // spread the bits evenly
        genga::radix_hist_kernel<<<nb, GENGA_SORT_THREADS, 0, st>>>(ka, N, shift, bits, nb, ctx->grp_counts, sb);
        genga::scan_kernel<<<1, 1024, 0, st>>>(ctx->grp_counts, (1 << bits) * nb);
        genga::radix_scatter_kernel<<<nb, GENGA_SORT_THREADS, 0, st>>>(ka, va, N, shift, bits, nb, ctx->grp_counts, kb, vb, sb);
        std::swap(ka, kb);
        std::swap(va, vb);
        shift += bits;
        ctx->launches += 3;
    }
    // ka, va: sorted.  kb is free: group-start flags, then their exclusive scan
    int* start = reinterpret_cast<int*>(kb);
    genga::group_mark_kernel<<<blocks, 256, 0, st>>>(ka, va, N, members, start);
    genga::scan_kernel<<<1, 1024, 0, st>>>(start, N);
    genga::group_offsets_kernel<<<blocks, 256, 0, st>>>(ka, start, N, offsets, summary);
    genga::group_max_kernel<<<std::min(blocks, 4 * ctx->num_sms), 256, 0, st>>>(offsets, summary, N);
    GK_CUDA(ctx, cudaGetLastError());
    ctx->launches += 4;
    return GENGA_KICK_OK;
}
