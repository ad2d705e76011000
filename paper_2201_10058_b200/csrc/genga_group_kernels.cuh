// sm_100a kernels of the grouping of close-encounter pairs into connected components
// (include/genga_group.h; App. A).
//
//   group_init_kernel   label[i] = i (every body its own tree), clears flags and the summary
//   group_hook_kernel   one thread per pair: lock-free union.  Invariant: label[x] <= x, and a root is
//                       only ever hooked under a SMALLER root (atomicCAS), so a tree's root is its
//                       smallest vertex whatever the order of the list
//   group_flat_kernel   label[i] -> root; group_of; sort key (root, or N for bodies in no pair)
//   (stable LSD radix sort of (key, body): the generic passes of genga_kick_sort.cuh)
//   group_mark_kernel / scan / group_offsets_kernel / group_max_kernel   members, offsets, summary
//
// Integer work only: every output is a fixed function of the pair SET.
// No code, header, table or helper is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace genga {

#define GENGA_STATUS_BAD_PAIR 16

__global__ void __launch_bounds__(256)
group_init_kernel(int* __restrict__ label, int* __restrict__ flag, int N, int* __restrict__ offsets, int* __restrict__ summary)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < N) { label[i] = i; flag[i] = 0; }
    if (i < 4) summary[i] = 0;
    if (i == 0) offsets[0] = 0;
}

// Root of x, with path halving.  The walk reads through L1 (ld.ca): the top of a large tree is read by
// every thread of the device, and L2-only reads of that one line serialise (measured on the 33,297-body
// group of config 3: 0.55 ms with ld.cg, 0.18 ms with ld.ca, one pass over all pairs).  A stale line is harmless: label[.] only ever
// moves to a proper ancestor, so a stale value is still an ancestor, and a stale "root" is caught by the
// atomicCAS of the hook, which returns the true parent and continues from there with a strictly smaller
// vertex.
__device__ __forceinline__ int group_find(int* label, int x)
{
    int p = __ldca(label + x);
    while (p != x) {
        const int gp = __ldca(label + p);
        if (gp != p) label[x] = gp;                         // still an ancestor: label[.] only ever decreases along a path
        x = p;
        p = gp;
    }
    return x;
}

__global__ void __launch_bounds__(256)
group_hook_kernel(const int2* __restrict__ pairs, const int* __restrict__ n_pairs, long long pair_rows, int N,
                  int sample, bool sampled, int* __restrict__ label, int* __restrict__ flag, int* __restrict__ summary,
                  int* __restrict__ status, int clip_status)
{
    // Two passes (host): first every `sample`-th pair (sampled = true), which already links most of a large
    // group; then, after group_compress_kernel has flattened the trees, the other pairs (sampled = false) --
    // for almost all of them both ends then point at the same root and the pair costs two cached reads.
    const long long total = min((long long)max(*n_pairs, 0), pair_rows);
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        summary[3] = (int)total;
        // a composed step (genga_hybrid_step) must not lose encounter pairs silently: clip_status = LIST_CLIPPED there
        if (clip_status && (long long)*n_pairs > pair_rows) atomicOr(status, clip_status);
    }
    for (long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x; p < total; p += (long long)gridDim.x * blockDim.x) {
        if (((p % sample) == 0) != sampled) continue;
        const int2 e = pairs[p];
        if (e.x < 0 || e.y < 0 || e.x >= N || e.y >= N) { atomicOr(status, GENGA_STATUS_BAD_PAIR); continue; }
        flag[e.x] = 1;
        flag[e.y] = 1;
        int ru = group_find(label, e.x), rv = group_find(label, e.y);
        while (ru != rv) {
            const int hi = max(ru, rv), lo = min(ru, rv);
            const int old = atomicCAS(label + hi, hi, lo);
            if (old == hi) break;                           // hi was a root and now hangs under lo
            ru = group_find(label, old);                    // hi had been hooked meanwhile: go on from there
            rv = group_find(label, lo);
        }
    }
}

// label[i] = root of i for every body (between the two hook passes)
__global__ void __launch_bounds__(256) group_compress_kernel(int* __restrict__ label, int N)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    int x = i, p = __ldcg(label + x);
    while (p != x) { x = p; p = __ldcg(label + x); }
    label[i] = x;                                           // an ancestor of i: concurrent readers stay correct
}

__global__ void __launch_bounds__(256)
group_flat_kernel(int* __restrict__ label, const int* __restrict__ flag, int N, int* __restrict__ group_of,
                  unsigned* __restrict__ keys, int* __restrict__ vals)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    int x = i, p = __ldcg(label + x);
    while (p != x) { x = p; p = __ldcg(label + x); }        // the trees are final: read only
    const bool in = flag[i] != 0;
    group_of[i] = in ? x : -1;
    keys[i] = in ? (unsigned)x : (unsigned)N;               // bodies in no pair sort behind every group
    vals[i] = i;
}

// sorted (key, body): members, group starts
__global__ void __launch_bounds__(256)
group_mark_kernel(const unsigned* __restrict__ keys, const int* __restrict__ vals, int N, int* __restrict__ members,
                  int* __restrict__ start)
{
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= N) return;
    const unsigned k = keys[p];
    const bool in = k != (unsigned)N;
    if (in) members[p] = vals[p];
    start[p] = in && (p == 0 || keys[p - 1] != k) ? 1 : 0;
}

// gidx = exclusive scan of the start flags
__global__ void __launch_bounds__(256)
group_offsets_kernel(const unsigned* __restrict__ keys, const int* __restrict__ gidx, int N, int* __restrict__ offsets,
                     int* __restrict__ summary)
{
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= N) return;
    const unsigned k = keys[p];
    if (k == (unsigned)N) return;
    const bool first = p == 0 || keys[p - 1] != k;
    if (first) offsets[gidx[p]] = p;
    if (p == N - 1 || keys[p + 1] == (unsigned)N) {          // the last body that is in a group
        const int ng = gidx[p] + (first ? 1 : 0);
        summary[0] = ng;
        summary[1] = p + 1;
        offsets[ng] = p + 1;
    }
}

__global__ void __launch_bounds__(256)
group_max_kernel(const int* __restrict__ offsets, int* __restrict__ summary, int N)
{
    const int ng = summary[0];
    int m = 0;
    for (int g = blockIdx.x * blockDim.x + threadIdx.x; g < ng; g += gridDim.x * blockDim.x)
        m = max(m, offsets[g + 1] - offsets[g]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0 && m > 0) atomicMax(summary + 2, m);       // a maximum: order-free
}

}  // namespace genga
