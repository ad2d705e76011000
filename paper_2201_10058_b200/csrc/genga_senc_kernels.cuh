// Kernels of include/genga_senc.h: close-encounter detection after the drift (App. A; DESIGN.md
// reading G16) and the small list kernels the SEnc recursion needs around genga_kick_list /
// genga_rcrit_list / genga_fg_list / genga_group / genga_bs.  Compiled with --fmad=false: every product and sum below
// rounds separately, in the order written (the detection's decision is an integer taken from floating point).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define GENGA_SENC_THREADS 256
#define GENGA_STATUS_BAD_DETECT_PAIR 16      // = GENGA_KICK_STATUS_BAD_PAIR
#define GENGA_STATUS_LIST_CLIPPED 128        // = GENGA_KICK_STATUS_LIST_CLIPPED

namespace genga {

// Minimum over tau in [0, 1] of the cubic p with p(0) = d0, p'(0) = m0, p(1) = d1, p'(1) = m1:
// p = a tau^3 + b tau^2 + c tau + d0; the root of p' with p'' >= 0 is (-b + sqrt(b^2 - 3ac)) / (3a), taken as
// -c / (b + sqrt(..)) for b > 0 (no cancellation when a -> 0: nearly uniform relative motion).
__device__ __forceinline__ double hermite_min(double d0, double m0, double d1, double m1)
{
    const double a = ((2.0 * d0 - 2.0 * d1) + m0) + m1;
    const double b = ((3.0 * d1 - 3.0 * d0) - 2.0 * m0) - m1;
    const double c = m0;
    double dmin = d0 <= d1 ? d0 : d1;
    const double disc = b * b - (3.0 * a) * c;
    if (disc >= 0.0) {
        const double s = sqrt(disc);
        double tau = -1.0;
        if (b > 0.0) tau = -c / (b + s);
        else if (a != 0.0) tau = (s - b) / (3.0 * a);
        if (tau > 0.0 && tau < 1.0) {
            const double p = ((a * tau + b) * tau + c) * tau + d0;
            if (p < dmin) dmin = p;
        }
    }
    return dmin;
}

// One thread per candidate; ballot/popc compaction with one atomic per warp on the total (rows beyond the capacity are
// counted, not written); per-body counts by integer atomics (order-free, so out_npairs is a fixed function of the input).
__global__ void __launch_bounds__(GENGA_SENC_THREADS)
detect_kernel(const double* __restrict__ pos0, const double* __restrict__ vel0, const double* __restrict__ pos1,
              const double* __restrict__ vel1, const double* __restrict__ rc_row, double f, double h, long long N,
              const int2* __restrict__ in_pairs, const int* __restrict__ in_n, long long in_rows,
              int2* __restrict__ out_pairs, long long cap, int* __restrict__ out_npairs, int* __restrict__ status)
{
    const long long count = min((long long)max(*in_n, 0), in_rows);
    const int lane = threadIdx.x & 31;
    const long long stride = (long long)gridDim.x * GENGA_SENC_THREADS;
    for (long long q = (long long)blockIdx.x * GENGA_SENC_THREADS + threadIdx.x; q - lane < count; q += stride) {
        bool enc = false;
        int i = 0, j = 0;
        if (q < count) {
            const int2 pr = in_pairs[q];
            i = pr.x; j = pr.y;
            if (i < 0 || j < 0 || i >= N || j >= N || i == j) {
                atomicOr(status, GENGA_STATUS_BAD_DETECT_PAIR);
            } else {
                double d[2], m[2];
#pragma unroll
                for (int s = 0; s < 2; s++) {
                    const double* P = s ? pos1 : pos0;
                    const double* V = s ? vel1 : vel0;
                    const double dx = P[j] - P[i], dy = P[N + j] - P[N + i], dz = P[2 * N + j] - P[2 * N + i];
                    const double ux = V[j] - V[i], uy = V[N + j] - V[N + i], uz = V[2 * N + j] - V[2 * N + i];
                    d[s] = dx * dx + dy * dy + dz * dz;
                    m[s] = h * (2.0 * (dx * ux + dy * uy + dz * uz));
                }
                const double dm = hermite_min(d[0], m[0], d[1], m[1]);
                const double ri = rc_row[i], rj = rc_row[j];
                const double R = f * (ri >= rj ? ri : rj);
                enc = dm < R * R;
            }
        }
        const unsigned mask = __ballot_sync(0xffffffffu, enc);
        if (mask) {
            int base = 0;
            if (lane == 0) base = atomicAdd(out_npairs + N, __popc(mask));
            base = __shfl_sync(0xffffffffu, base, 0);
            if (enc) {
                const long long slot = (long long)base + __popc(mask & ((1u << lane) - 1u));
                if (slot < cap) out_pairs[slot] = i < j ? make_int2(i, j) : make_int2(j, i);
                atomicAdd(out_npairs + i, 1);
                atomicAdd(out_npairs + j, 1);
            }
        }
    }
}

// dst[.][i] = src[.][i] for the bodies of a list (state saved before a level's drift / restored for the level below)
__global__ void __launch_bounds__(GENGA_SENC_THREADS)
copy_list_kernel(double* __restrict__ dst_pos, double* __restrict__ dst_vel, const double* __restrict__ src_pos,
                 const double* __restrict__ src_vel, long long N, const int* __restrict__ list,
                 const int* __restrict__ n_list, long long list_rows)
{
    const long long count = min((long long)max(*n_list, 0), list_rows);
    for (long long q = (long long)blockIdx.x * GENGA_SENC_THREADS + threadIdx.x; q < count;
         q += (long long)gridDim.x * GENGA_SENC_THREADS) {
        const long long i = list[q];
        if (i < 0 || i >= N) continue;
#pragma unroll
        for (int c = 0; c < 3; c++) {
            dst_pos[c * N + i] = src_pos[c * N + i];
            dst_vel[c * N + i] = src_vel[c * N + i];
        }
    }
}

// per-level statistics of one sub-step: candidates, close-encounter pairs, and (deepest level) groups / bodies of the
// Bulirsch-Stoer phase
__global__ void senc_stats_kernel(int* __restrict__ stats, const int* __restrict__ n_cand, const int* __restrict__ n_enc,
                                  const int* __restrict__ summary, int bs_level, long long cap, int* __restrict__ status)
{
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        // a list longer than the pair capacity was clipped: the levels below saw only part of the encounters
        if (*n_cand > cap || *n_enc > cap) atomicOr(status, GENGA_STATUS_LIST_CLIPPED);
        if (stats) {
            stats[0] += *n_cand;
            stats[1] += *n_enc;
            if (bs_level) { stats[2] += summary[0]; stats[3] += summary[1]; }
        }
    }
}

}  // namespace genga
