// sm_100a kernels of the Bulirsch-Stoer integration of close-encounter groups (include/genga_bs.h;
// PAPER.md:47, :559-597, App. A), in three regimes of one template:
//   bs_kernel<WARP>   one WARP per group of up to 8 bodies, one lane per body, eight groups side by side in a CTA, the
//                     group's state in the warp's slice of shared memory, no CTA-wide barrier -- nearly all groups are
//                     pairs;
//   bs_kernel<CTA>    one CTA per group of 9 .. 32 bodies, eight lanes per body; with the warp regime the regime BS-B
//                     of Table 2 (sec. 6.1.1: n <= 32);
//   bs_cluster_kernel one thread-block CLUSTER of 8 CTAs x 256 threads per group of 33 .. 256 bodies, eight lanes per
//                     body: the CTAs publish their 32 bodies' positions in their own shared memory, gather the others'
//                     through distributed shared memory and meet at one cluster barrier per force evaluation; many
//                     clusters side by side: the regime BS-A of Table 2;
//   bs_kernel<COOP>   ONE group at a time over the whole grid (cooperative launch, 64-thread CTAs): the paper's
//                     BS-M regime ("distributed over multiple thread blocks ... sub-steps ...
//                     controlled from the host ... many different kernel calls") -- but here the sub-steps stay
//                     on the device: positions are exchanged through L2 (double-buffered) and the CTAs meet at
//                     one grid-wide barrier per force evaluation.  Groups of 257 .. grid size bodies.
//
// The scheme is the textbook Gragg-Bulirsch-Stoer method fixed as reading G15 in DESIGN.md: modified
// midpoint with n_k = 2k sub-steps (k = 1..8), Aitken-Neville extrapolation in h^2, relative error per body
// (Euclidean norms of position and of velocity), the whole group advancing synchronously with one step
// size.  Every operation is written in the order of that description and the build forbids contraction
// (--fmad=false), the force sum runs over the group's members in list order: the result is a fixed
// function of the inputs.
//
// No code, header, table or helper is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <cooperative_groups.h>

namespace genga {

#define GENGA_BS_MODE_CTA 0
#define GENGA_BS_MODE_COOP 1
#define GENGA_BS_MODE_WARP 2
#define GENGA_BS_MODE_CLUSTER 3
#define GENGA_BS_CLUSTER 8              // CTAs of a cluster (the portable maximum)
#define GENGA_BS_CLUSTER_BODIES 32      // bodies per CTA of a cluster = GENGA_BS_THREADS / GENGA_BS_SUB
#define GENGA_BS_WARP_MAX 32            // rows of a warp's shared-memory slice
#define GENGA_BS_SEQ_MAX 8              // largest group of the warp-per-group regime (force sum in member order)
#define GENGA_BS_CTA_MAX 32             // largest group of the one-CTA regime = GENGA_BS_THREADS / GENGA_BS_SUB
#define GENGA_BS_THREADS 256            // CTA of the one-CTA-per-group regime = largest group it takes
#define GENGA_BS_COOP_THREADS 256       // CTA of the whole-grid regime (its bodies' lists are pooled: bs_build_lists)
#define GENGA_BS_SUB 8                  // whole-grid regime: lanes per body, each summing the terms with j = lane (mod 8)
                                        // (groups too large for that: one lane per body, the same eight partial sums)
#define GENGA_BS_TILE 256               // j-bodies staged per round in the whole-grid regime
#define GENGA_BS_TEAM_CTAS 16           // whole-grid regime in teams: CTAs of the small teams (512 bodies at eight lanes each)
#define GENGA_BS_KMAX 8
#define GENGA_BS_MAX_LEVELS 4
#define GENGA_BS_MAX_HALVINGS 60
#define GENGA_STATUS_GROUP_TOO_LARGE 32
#define GENGA_STATUS_BS_NOT_CONVERGED 64
#define GENGA_STATUS_BS_LIST_ESCAPE 512

// the changeover function K (reading G1), IEEE operations in a fixed order
__device__ __forceinline__ double bs_K(double r, double rc)
{
    const double y = (r - 0.1 * rc) / (0.9 * rc);
    if (y <= 0.0) return 0.0;
    if (y >= 1.0) return 1.0;
    return (y * y) / (2.0 * y * y - 2.0 * y + 1.0);
}

// Scratch of the whole-grid regime (device memory, library-owned): the group's positions in two buffers
// (force evaluation e publishes into buffer e & 1 while slower CTAs may still read the other one), G m,
// the critical-radius rows, and four slots for the group-wide error maximum.
struct BsGlobal {
    double* x[2]; double* y[2]; double* z[2];
    double2* pk[2];                     // the same positions packed with the far-pair bound: (x, y), (z, bound) per body,
                                        // one 32-byte sector per list entry
    double2* sr;                        // what a NEAR list entry needs besides: (G m, rc0), (rc1, rc2), (rc3, -) per body
    double* gm;
    double* rcsq;                       // far-pair bound of each body (bs_far_bound)
    double* rc[GENGA_BS_MAX_LEVELS];
    // neighbour lists of the whole-grid regime (bs_build_lists)
    double* lr;                         // [n] sqrt(far-pair bound) of each body
    double* la;                         // [n] A_b: bound on its deviation from straight-line motion during the call
    double* ld;                         // [n] |v_b| |dt| + A_b: bound on its displacement (cheap first test)
    double* vx; double* vy; double* vz; // [n] velocities at the start of the call
    int* nbr;                           // the warps' lists: chunks of 32 entries, bs_chunk_words(nlevels) 8-byte words each
    long long nbr_capacity;             // ... its size in 4-byte units
    unsigned long long* cursor;         // entries reserved so far (zero between groups)
    unsigned long long* err;            // [4], all zero between uses
    // teams: the co-resident grid cut into teams of team_ctas CTAs, each integrating its own groups with a barrier
    // of its own (0: one team = the whole grid, cooperative-groups barrier).  bs_run points the arrays above at the
    // team's slice of the scratch; ctrl = [teams][16] words: err[4], cursor, barrier counter.
    int team_ctas;
    int tb;                             // this CTA's index within its team (set by bs_run)
    unsigned long long* bar;            // the team's barrier counter (only ever incremented within a launch)
    // diagnostics of the step-size control (include/genga_bs.h: genga_bs_set_stats, genga_bs_totals)
    unsigned long long* totals;         // [4] accepted macro steps, rejected attempts, force evaluations, groups: summed
    int4* stats;                        // [stats_rows] per group (accepted, rejected, force evaluations, bodies), or nullptr
    long long stats_rows;
};

// shared memory: one-CTA regime: the whole group; whole-grid regime: one tile of j-bodies
template <int ROWS>
struct BsShared {
    double x[ROWS], y[ROWS], z[ROWS], gm[ROWS];
    double rcsq[ROWS];                  // far-pair bound of each body (bs_far_bound)
    double rc[GENGA_BS_MAX_LEVELS][ROWS];
    double red[8];
    double errmax;
    // cluster regime: this CTA's bodies, published for the other CTAs of the cluster (two buffers: force evaluation e
    // publishes into buffer e & 1 while slower CTAs may still gather from the other one), and its error maxima
    double pubx[2][GENGA_BS_CLUSTER_BODIES], puby[2][GENGA_BS_CLUSTER_BODIES], pubz[2][GENGA_BS_CLUSTER_BODIES];
    double emax[2];
    unsigned long long bar_target;      // whole-grid regime in teams: the count the team's barrier has to reach next
};

// Barrier over the CTAs that integrate a group together: the whole grid (cooperative groups), or one team of it -- the
// CTAs of a cooperative launch are co-resident, so a team may wait on a counter of its own: every CTA adds one and
// waits until all team_ctas have (the counter is never reset within a launch; each CTA keeps the next target).
template <int ROWS>
__device__ __forceinline__ void bs_gsync(BsShared<ROWS>& S, const BsGlobal& Gm)
{
    // (the whole grid is one team of gridDim.x CTAs.  The poll is a RELAXED load followed by one fence: an acquire load,
    // like the one in cooperative groups' grid barrier, invalidates the SM's L1 on every iteration -- and with it the
    // extrapolation tableaus, in local memory, of the CTAs that are still working)
    __syncthreads();
    if (threadIdx.x == 0) {
        S.bar_target += (unsigned long long)Gm.team_ctas;
        __threadfence();
        atomicAdd(Gm.bar, 1ULL);
        unsigned long long seen;
        do {
            asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(seen) : "l"(Gm.bar) : "memory");
        } while (seen < S.bar_target);
        __threadfence();
    }
    __syncthreads();
}

// A pair with r^2 >= max(bound_i, bound_j), bound_b = rc0_b^2 (1 + 2^-20), has r > rc0_ij by more than 2^-22 relative:
// y = (r - 0.1 rc)/(0.9 rc) > 1 whatever its rounding, K_0 = 1 and W_BS = prod (1 - K_k) = 0 EXACTLY -- the pair adds
// nothing, as in the definition, and costs 8 FP64 instructions instead of ~100 (sqrt, a divide per level and one for
// the term).  In the large groups of a disk almost all pairs are of this kind: a group is a chain of neighbours.
__device__ __forceinline__ double bs_far_bound(double rc0) { return (rc0 * rc0) * (1.0 + 9.5367431640625e-07); }

// The weight and the factor of a pair inside a far-pair bound: s = G m_j prod_k (1 - K(r; max(rc_k,i, rc_k,j))) / r^3;
// false: the product is 0 and the pair adds nothing.  OUT OF LINE, one copy per kernel: a square root, a divide for s and
// two per level are ~400 instructions, and the force loops name a pair in up to a dozen places (lanes' sub-lists x
// loads in flight, all-pairs fallback) -- inlined, the whole-grid kernels were 13,000 - 61,000 instructions long and
// their list walk ran out of the instruction cache (12 us per near pair; profiles/ncu_r02c.md).
__device__ __forceinline__ bool bs_pair_factor_inline(double r2, double gmj, int nlevels, double rci0, double rci1, double rci2,
                                                      double rci3, double rcj0, double rcj1, double rcj2, double rcj3, double& s)
{
    const double r = sqrt(r2);
    double W = 1.0;
    W *= (1.0 - bs_K(r, fmax(rci0, rcj0)));
    if (1 < nlevels) W *= (1.0 - bs_K(r, fmax(rci1, rcj1)));
    if (2 < nlevels) W *= (1.0 - bs_K(r, fmax(rci2, rcj2)));
    if (3 < nlevels) W *= (1.0 - bs_K(r, fmax(rci3, rcj3)));
    if (W == 0.0) return false;
    s = gmj * W / (r2 * r);
    return true;
}
// (the whole-grid kernels, which name a pair in the all-pairs fallback of every lane count, take it out of line; the warp,
// CTA and cluster regimes, each with one pair loop, inline it)
__device__ __noinline__ bool bs_pair_factor(double r2, double gmj, int nlevels, double rci0, double rci1, double rci2, double rci3,
                                            double rcj0, double rcj1, double rcj2, double rcj3, double& s)
{
    return bs_pair_factor_inline(r2, gmj, nlevels, rci0, rci1, rci2, rci3, rcj0, rcj1, rcj2, rcj3, s);
}

// one pair term of dv_i/dt, added in place: G m_j prod_k (1 - K(r; max(rc_k,i, rc_k,j))) (q_j - q_i) / r^3.
// Test-particle modes (sec. 8.1, Fig. 14): a semi-active particle j is staged with the SIGN BIT of
// G m_j set; it acts on nobody in TP 1 and on the massive bodies only in TP 2 (particles never feel each other).
#define GENGA_BS_PAIR(XJ, YJ, ZJ, GMJ, RCJ, BNDJ) GENGA_BS_PAIR_ACC(XJ, YJ, ZJ, GMJ, RCJ, BNDJ, ax, ay, az)
#define GENGA_BS_PAIR_ACC(XJ, YJ, ZJ, GMJ, RCJ, BNDJ, AX, AY, AZ)                                      \
    {                                                                                                  \
        double gmj = (GMJ);                                                                            \
        bool skip = false;                                                                             \
        if (__double2hiint(gmj) < 0) { skip = i_tp || tp_mode != 2; gmj = -gmj; }                      \
        const double dx = (XJ) - x, dy = (YJ) - y, dz = (ZJ) - z;                                      \
        const double r2 = dx * dx + dy * dy + dz * dz;                                                 \
        if (!skip && r2 < fmax(bnd_i, (BNDJ))) {                                                       \
            double s;                                                                                  \
            if (MODE == GENGA_BS_MODE_COOP                                                             \
                    ? bs_pair_factor(r2, gmj, nlevels, rci[0], rci[1], rci[2], rci[3], RCJ(0),         \
                                     1 < nlevels ? RCJ(1) : 0.0, 2 < nlevels ? RCJ(2) : 0.0,           \
                                     3 < nlevels ? RCJ(3) : 0.0, s)                                    \
                    : bs_pair_factor_inline(r2, gmj, nlevels, rci[0], rci[1], rci[2], rci[3], RCJ(0),  \
                                            1 < nlevels ? RCJ(1) : 0.0, 2 < nlevels ? RCJ(2) : 0.0,    \
                                            3 < nlevels ? RCJ(3) : 0.0, s)) {                          \
                AX = AX + s * dx; AY = AY + s * dy; AZ = AZ + s * dz;                                  \
            }                                                                                          \
        }                                                                                              \
    }

// ---------------------------------------------------------------------------------------------------------------------
// Neighbour lists of the whole-grid regime.  A large group of a disk is a chain of neighbours: of its n^2 pairs all but
// a few per body lie far outside every critical radius for the whole call and add exactly nothing (bs_far_bound).  At
// the start of a group every lane lists the partners it may ever have to evaluate: those whose STRAIGHT-LINE relative
// motion over the call comes closer than the far-pair radius plus the two bodies' allowances,
//     min over tau in [0, dt] of |dq_ij(t0) + dv_ij(t0) tau|  <  max(R_i, R_j) + A_i + A_j,
//     R_b = sqrt(far-pair bound of b),    A_b = G m_star dt^2 / |q_b(t0)|^2   (twice the Sun's a dt^2 / 2)
// A_b bounds the body's deviation from q_b(t0) + v_b(t0) tau during the call; every force evaluation CHECKS it (it
// knows its time tau) and raises GENGA_STATUS_BS_LIST_ESCAPE if a body strayed further -- then, and only then, a pair
// outside the lists may have come inside a critical radius unseen.  A pair outside the lists therefore has
// r > max(R_i, R_j) at every force evaluation and contributes exactly 0, as in the all-pairs sum: the lists change the
// cost (n x a few partners instead of n^2 pairs per force evaluation) and the ORDER of the sum (below), nothing else.
//
// The lists are kept per WARP, not per lane: the entries of the warp's bodies (32 / SUB of them), sorted by body, in
// chunks of 32.  A force evaluation walks the chunks with all 32 lanes -- one entry per lane whatever body it belongs
// to, so that a body with 100 partners and one with 5 cost the warp the same per entry (per-lane lists left a warp
// waiting for its longest lane, 9 of 32 lanes active on average in the dense group of configs[3] at 2 levels x 2
// sub-steps: profiles/ncu_r02c.md) -- and adds the terms of a chunk with a segmented scan over the lanes (segments =
// bodies; IEEE additions in a fixed tree), the segment sums to the bodies' accumulators in chunk order.  The order of a
// body's sum is thus a fixed function of the list, i.e. of the inputs; it is the kernel's own choice
// like every force-sum order here (reading G15).
// Lists that do not fit the scratch (nbr_capacity) are not used: that group falls back to all pairs.
// ---------------------------------------------------------------------------------------------------------------------
template <int NL>
struct BsList {
    bool on;                            // lists in use for this group (team-uniform)
    long long cbase;                    // this CTA's list: first chunk (CTA-uniform) ...
    int cchunks;                        // ... and number of chunks of 32 entries
    double q0[3], v0[3];                // the body's state at the start of the call
    double a2;                          // A_b^2
    double gmi;                         // G m_b (published with the position: what a partner's walk needs of this body)
};

// A chunk of a CTA's list: 32 entries, field by field (every load of the walk is one coalesced 256-byte row):
//   row 0       (j, slot) -- the partner's position within the group (-1: padding) and which of the CTA's bodies the
//               entry belongs to (thread / SUB of its lanes); the entries of a CTA are sorted by slot
//   row 1       max(bound_i, bound_j), the far-pair bound of the pair (bs_far_bound)
//   row 2 + k   1 / (0.9 max(rc_k,i, rc_k,j)), k < nlevels: y_k = r / (0.9 rc) - 1/9 (bs_pair_factor_listed)
// i.e. everything about the pair that does not change during the call: a force evaluation reads the entry and ONE
// 32-byte record of the partner, (x, y), (z, G m), at its current position.
__device__ __forceinline__ int bs_chunk_words(int nlevels) { return 32 * (2 + nlevels); }

// The factor s = G m_j prod_k (1 - K(r; rc_k)) / r^3 of a listed pair inside its far-pair bound, with the quantities
// the list holds.  1 - K(y) = (1 - y)^2 / (2 y^2 - 2 y + 1) (reading G1), so the product over the
// levels is one quotient; 1/r comes from the MUFU.RSQ64H seed and a third-order correction (relative error < 2^-58), the
// reciprocal of the denominator from the MUFU.RCP64H seed and two Newton steps: ~35 FP64 instructions where the
// literal evaluation (a square root, two divisions per level, one for the term) takes ~450.  The same function of
// (r, rc_k) as bs_K up to a few units in the last place of each factor -- the whole-grid regime's force sum differs
// from the oracle's by its order already (reading G15); the parity bound of tests/test_gpu_bs.py has room for 1e-12.
// false: some level has y_k >= 1, the pair adds nothing.
__device__ __forceinline__ bool bs_pair_factor_listed(double r2, double gmj, int nlevels, double b0, double b1, double b2,
                                                      double b3, double& s)
{
    double y0;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y0) : "d"(r2));
    const double e = fma(-r2, y0 * y0, 1.0);
    const double rinv = y0 * fma(e, fma(0.375, e, 0.5), 1.0);
    const double r = r2 * rinv;
    double num = 1.0, den = 1.0;
    const double bk[GENGA_BS_MAX_LEVELS] = {b0, b1, b2, b3};
#pragma unroll
    for (int k = 0; k < GENGA_BS_MAX_LEVELS; k++)
        if (k < nlevels) {
            const double y = fma(r, bk[k], -0.1111111111111111);
            if (y >= 1.0) return false;
            if (y > 0.0) {
                const double omy = 1.0 - y;
                num = num * (omy * omy);
                den = den * fma(2.0 * y, y - 1.0, 1.0);
            }
        }
    double x;                                                   // 1 / den, den in (2^-4, 1]
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(x) : "d"(den));
    x = fma(x, fma(-den, x, 1.0), x);
    x = fma(x, fma(-den, x, 1.0), x);
    s = ((gmj * num) * x) * ((rinv * rinv) * rinv);
    return true;
}

// Every thread publishes the position of its body i (if i < n) and gets dv_i/dt back:
//   - G m_star q / |q|^3 + the pair terms over j = 0 .. n-1, j != i, in that order.
// COOP: `eval` counts the force evaluations of the group (buffer parity); one grid barrier per call.
template <int MODE>
__device__ __forceinline__ void bs_sync()
{
    if (MODE == GENGA_BS_MODE_WARP) __syncwarp(); else __syncthreads();
}

template <int MODE, int ROWS, int SUB>
__device__ __forceinline__ void bs_force(BsShared<ROWS>& S, const BsGlobal& Gm, int& eval, int i, int n, int nlevels,
                                         bool i_tp, int tp_mode, double mu, const double (&rci)[GENGA_BS_MAX_LEVELS], const double (&q)[3],
                                         double (&a)[3], const BsList<8 / SUB>& L, double tau, int* __restrict__ status)
{
    const double bnd_i = bs_far_bound(rci[0]);
    const double x = q[0], y = q[1], z = q[2];
    const double r2s = x * x + y * y + z * z;
    const double rs = sqrt(r2s);
    const double s0 = -mu / (r2s * rs);
    double ax = s0 * x, ay = s0 * y, az = s0 * z;
    constexpr bool COOP = MODE == GENGA_BS_MODE_COOP;
    if constexpr (MODE == GENGA_BS_MODE_WARP) {
        bs_sync<MODE>();                                      // the previous readers are done
        if (i < n) { S.x[i] = x; S.y[i] = y; S.z[i] = z; }
        bs_sync<MODE>();
        if (i < n) {
#define GENGA_BS_RCJ(k) S.rc[k][j]
            for (int j = 0; j < n; j++) {
                if (j == i) continue;
                GENGA_BS_PAIR(S.x[j], S.y[j], S.z[j], S.gm[j], GENGA_BS_RCJ, S.rcsq[j])
            }
#undef GENGA_BS_RCJ
        }
    } else if constexpr (MODE == GENGA_BS_MODE_CTA) {
        // Eight lanes per body inside one CTA (groups of up to 32 bodies): the eight partial sums and the tree as below.
        const int sub = threadIdx.x & (SUB - 1);
        __syncthreads();                                      // the previous readers are done
        if (i < n && sub == 0) { S.x[i] = x; S.y[i] = y; S.z[i] = z; }
        __syncthreads();
        const double sx = ax, sy = ay, sz = az;
        ax = 0.0; ay = 0.0; az = 0.0;
        if (i < n) {
#define GENGA_BS_RCJ(k) S.rc[k][jj]
            for (int jj = sub; jj < n; jj += SUB) {
                if (jj == i) continue;
                GENGA_BS_PAIR(S.x[jj], S.y[jj], S.z[jj], S.gm[jj], GENGA_BS_RCJ, S.rcsq[jj])
            }
#undef GENGA_BS_RCJ
        }
#pragma unroll
        for (int o = 1; o < SUB; o <<= 1) {
            ax = ax + __shfl_xor_sync(0xffffffffu, ax, o);
            ay = ay + __shfl_xor_sync(0xffffffffu, ay, o);
            az = az + __shfl_xor_sync(0xffffffffu, az, o);
        }
        ax = sx + ax; ay = sy + ay; az = sz + az;
    } else if constexpr (MODE == GENGA_BS_MODE_CLUSTER) {
        // Eight lanes per body (as below), the group spread over the CTAs of a cluster: publish, one cluster barrier,
        // gather everybody's positions through distributed shared memory, then sum from the local copy.
        cooperative_groups::cluster_group cl = cooperative_groups::this_cluster();
        const int p = eval & 1;
        eval++;
        const int t = threadIdx.x, sub = t & (SUB - 1);
        if (i < n && sub == 0) { S.pubx[p][t / SUB] = x; S.puby[p][t / SUB] = y; S.pubz[p][t / SUB] = z; }
        cl.sync();
        for (int idx = t; idx < n; idx += ROWS) {
            const unsigned r = idx / GENGA_BS_CLUSTER_BODIES, o = idx % GENGA_BS_CLUSTER_BODIES;
            S.x[idx] = cl.map_shared_rank(&S.pubx[p][0], r)[o];
            S.y[idx] = cl.map_shared_rank(&S.puby[p][0], r)[o];
            S.z[idx] = cl.map_shared_rank(&S.pubz[p][0], r)[o];
        }
        __syncthreads();
        const double sx = ax, sy = ay, sz = az;
        ax = 0.0; ay = 0.0; az = 0.0;
        if (i < n) {
#define GENGA_BS_RCJ(k) S.rc[k][jj]
            for (int jj = sub; jj < n; jj += SUB) {
                if (jj == i) continue;
                GENGA_BS_PAIR(S.x[jj], S.y[jj], S.z[jj], S.gm[jj], GENGA_BS_RCJ, S.rcsq[jj])
            }
#undef GENGA_BS_RCJ
        }
#pragma unroll
        for (int o = 1; o < SUB; o <<= 1) {
            ax = ax + __shfl_xor_sync(0xffffffffu, ax, o);
            ay = ay + __shfl_xor_sync(0xffffffffu, ay, o);
            az = az + __shfl_xor_sync(0xffffffffu, az, o);
        }
        ax = sx + ax; ay = sy + ay; az = sz + az;
    } else {
        // The pair terms with j = s (mod 8) are summed in ascending j from 0 into p_s, s = 0 .. 7; the eight partial
        // sums are combined as ((p0 + p1) + (p2 + p3)) + ((p4 + p5) + (p6 + p7)) and added to the Sun term.
        //   SUB = 8: eight lanes per body, lane `sub` holds p_sub, xor butterfly (IEEE addition commutes, so every
        //            lane of the octet gets the same bits);
        //   SUB = 1: one lane per body holds all eight (groups too large for eight lanes each) -- same arithmetic.
        const int p = eval & 1;
        eval++;
        const int t = threadIdx.x, sub = t & (SUB - 1);
        if (i < n && sub == 0) {
            Gm.x[p][i] = x; Gm.y[p][i] = y; Gm.z[p][i] = z;
            if (L.on) { Gm.pk[p][2 * i] = make_double2(x, y); Gm.pk[p][2 * i + 1] = make_double2(z, L.gmi); }
        }
        // the CTA's bodies, for the lanes that walk their entries: current positions and the accumulators
        constexpr int WB = GENGA_BS_COOP_THREADS / SUB, NW = GENGA_BS_COOP_THREADS / 32;
        __shared__ double wpos[WB][3];
        __shared__ double wacc[WB][3];
        __shared__ double wcarry[NW][3];                                // a warp's terms of the body its range starts inside
        __shared__ int wcarry_slot[NW];                                 // ... and which body that is (-1: none)
        const int lane = t & 31, wid = t >> 5;
        if (L.on) {
            if (sub == 0) {
                wpos[t / SUB][0] = x; wpos[t / SUB][1] = y; wpos[t / SUB][2] = z;
                wacc[t / SUB][0] = 0.0; wacc[t / SUB][1] = 0.0; wacc[t / SUB][2] = 0.0;
            }
            if (lane == 0) { wcarry[wid][0] = 0.0; wcarry[wid][1] = 0.0; wcarry[wid][2] = 0.0; wcarry_slot[wid] = -1; }
        }
        bs_gsync(S, Gm);
        const double sx = ax, sy = ay, sz = az;
        double px[8 / SUB], py[8 / SUB], pz[8 / SUB];
#pragma unroll
        for (int u = 0; u < 8 / SUB; u++) { px[u] = 0.0; py[u] = 0.0; pz[u] = 0.0; }
        if (L.on) {
            if (i < n) {
                // the body must still be where the lists allow it to be
                const double ex = x - (L.q0[0] + L.v0[0] * tau), ey = y - (L.q0[1] + L.v0[1] * tau), ez = z - (L.q0[2] + L.v0[2] * tau);
                if (ex * ex + ey * ey + ez * ez > L.a2) atomicOr(status, GENGA_STATUS_BS_LIST_ESCAPE);
            }
            // warp w walks the chunks [w C / 8, (w + 1) C / 8) of the CTA's list (sorted by body): the bodies of its range
            // are its own but for the first, which may have begun in the range of the warp before
            const int cw = bs_chunk_words(nlevels);
            const int c0 = (int)((long long)wid * L.cchunks / NW), c1 = (int)((long long)(wid + 1) * L.cchunks / NW);
            const unsigned long long* rec = reinterpret_cast<const unsigned long long*>(Gm.nbr) + (L.cbase + c0) * cw + lane;
            int prev_slot = -1;
            if (c0 > 0 && c1 > c0) prev_slot = (int)(__ldcg(rec - lane - cw + 31) >> 32);     // (warp-uniform)
            if (lane == 0) wcarry_slot[wid] = prev_slot;
            // Three chunks in flight: while chunk c is evaluated, the partners' records of chunk c + 1 are on their way
            // (their indices arrived during chunk c - 1) and so are the indices of chunk c + 2.  Two register sets take
            // the partners' records in turn (no copies between the stages).
            constexpr unsigned long long PAD = 0xffffffffULL | (0x7fffULL << 32);
            struct Stage { double bnd, b[GENGA_BS_MAX_LEVELS]; double2 pa, pb; };
            Stage s0, s1;
            s0.bnd = 0.0; s0.pa = make_double2(0.0, 0.0); s0.pb = s0.pa;
#pragma unroll
            for (int k = 0; k < GENGA_BS_MAX_LEVELS; k++) s0.b[k] = 0.0;
            s1 = s0;
            const double2* const pkp = Gm.pk[p];
            auto gather = [&](Stage& g, unsigned long long js, const unsigned long long* rb) {
                const int jb = (int)(unsigned)(js & 0xffffffffULL);
                if (jb >= 0) {
                    g.bnd = __longlong_as_double((long long)__ldcg(rb + 32));
#pragma unroll
                    for (int k = 0; k < GENGA_BS_MAX_LEVELS; k++)
                        if (k < nlevels) g.b[k] = __longlong_as_double((long long)__ldcg(rb + 64 + 32 * k));
                    g.pa = __ldcg(pkp + 2 * jb); g.pb = __ldcg(pkp + 2 * jb + 1);
                }
            };
            auto evaluate = [&](const Stage& g, unsigned long long js) {
                const int jj = (int)(unsigned)(js & 0xffffffffULL), slot = (int)(js >> 32);
                double tx = 0.0, ty = 0.0, tz = 0.0;
                if (jj >= 0) {
                    const double dx = g.pa.x - wpos[slot][0], dy = g.pa.y - wpos[slot][1], dz = g.pb.x - wpos[slot][2];
                    const double r2 = dx * dx + dy * dy + dz * dz;
                    double sfac;
                    if (r2 < g.bnd && bs_pair_factor_listed(r2, g.pb.y, nlevels, g.b[0], g.b[1], g.b[2], g.b[3], sfac)) {
                        tx = sfac * dx; ty = sfac * dy; tz = sfac * dz;
                    }
                }
                // sum of each body's terms of this chunk: inclusive scan over the lanes within runs of equal slot
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const int so = __shfl_up_sync(0xffffffffu, slot, o);
                    const double ux = __shfl_up_sync(0xffffffffu, tx, o), uy = __shfl_up_sync(0xffffffffu, ty, o),
                                 uz = __shfl_up_sync(0xffffffffu, tz, o);
                    const int take = (lane >= o && so == slot) ? 1 : 0;
                    asm("{\n\t.reg .pred q;\n\tsetp.ne.s32 q, %6, 0;\n\t@q add.rn.f64 %0, %3, %0;\n\t@q add.rn.f64 %1, %4, %1;\n\t"
                        "@q add.rn.f64 %2, %5, %2;\n\t}"
                        : "+d"(tx), "+d"(ty), "+d"(tz) : "d"(ux), "d"(uy), "d"(uz), "r"(take));
                }
                const int snext = __shfl_down_sync(0xffffffffu, slot, 1);
                if (slot < WB && (lane == 31 || snext != slot)) {      // the last lane of a run holds its sum
                    double* acc = slot == prev_slot ? wcarry[wid] : wacc[slot];
                    acc[0] = acc[0] + tx; acc[1] = acc[1] + ty; acc[2] = acc[2] + tz;
                }
                __syncwarp();                                           // the next chunk may continue the run in another lane
            };
            unsigned long long jsA = PAD, jsB = PAD, jsC = PAD;             // entries of chunk c + 2, c + 1, c
            const unsigned long long* rA = rec;                             // row 0 of the chunk jsA is loaded from next
            for (int c = c0 - 2; c < c1; c += 2) {
                jsC = jsB; jsB = jsA;
                jsA = c + 2 < c1 ? __ldcg(rA) : PAD;
                gather(s0, jsB, rA - cw);                                   // chunk c + 1
                if (c >= c0) evaluate(s1, jsC);                             // chunk c (warp-uniform condition)
                jsC = jsB; jsB = jsA;
                jsA = c + 3 < c1 ? __ldcg(rA + cw) : PAD;
                gather(s1, jsB, rA);                                        // chunk c + 2
                if (c + 1 >= c0 && c + 1 < c1) evaluate(s0, jsC);           // chunk c + 1
                rA += 2 * cw;
            }
            __syncthreads();
            // a body's sum: what the warp that met its first entry gathered, then the carries of the warps after it, in order
            px[0] = wacc[t / SUB][0]; py[0] = wacc[t / SUB][1]; pz[0] = wacc[t / SUB][2];
#pragma unroll
            for (int w = 1; w < NW; w++)
                if (wcarry_slot[w] == t / SUB) { px[0] = px[0] + wcarry[w][0]; py[0] = py[0] + wcarry[w][1]; pz[0] = pz[0] + wcarry[w][2]; }
            __syncthreads();                                            // (before the next evaluation clears them)
        }
        for (int j0 = 0; j0 < (L.on ? 0 : n); j0 += ROWS) {   // ROWS is a multiple of 8: (j0 + jj) mod 8 = jj mod 8
            __syncthreads();
            if (t < ROWS && j0 + t < n) {
                S.x[t] = __ldcg(Gm.x[p] + j0 + t); S.y[t] = __ldcg(Gm.y[p] + j0 + t); S.z[t] = __ldcg(Gm.z[p] + j0 + t);
                S.gm[t] = __ldcg(Gm.gm + j0 + t);
                S.rcsq[t] = __ldcg(Gm.rcsq + j0 + t);
                for (int k = 0; k < nlevels; k++) S.rc[k][t] = __ldcg(Gm.rc[k] + j0 + t);
            }
            __syncthreads();
            if (i < n) {
                const int m = min(ROWS, n - j0);
#define GENGA_BS_RCJ(k) S.rc[k][jj]
                for (int j8 = 0; j8 < m; j8 += 8) {
#pragma unroll
                    for (int u = 0; u < 8 / SUB; u++) {
                        const int jj = j8 + sub + SUB * u;    // this lane's residues j mod 8: sub, sub + SUB, ..
                        if (jj < m && j0 + jj != i) {
                            GENGA_BS_PAIR_ACC(S.x[jj], S.y[jj], S.z[jj], S.gm[jj], GENGA_BS_RCJ, S.rcsq[jj], px[u], py[u], pz[u])
                        }
                    }
                }
#undef GENGA_BS_RCJ
            }
        }
        // p_r = the terms with j = r (mod 8); lane `sub` holds p_sub, p_sub+SUB, ..: first the pairs of the tree that lie
        // in different lanes (xor butterfly: IEEE addition commutes, so every lane of the body gets the same bits),
        // then those within the lane: ((p0 + p1) + (p2 + p3)) + ((p4 + p5) + (p6 + p7)) whatever SUB is
        if (!L.on) {
#pragma unroll
        for (int o = 1; o < SUB; o <<= 1) {
#pragma unroll
            for (int u = 0; u < 8 / SUB; u++) {
                px[u] = px[u] + __shfl_xor_sync(0xffffffffu, px[u], o);
                py[u] = py[u] + __shfl_xor_sync(0xffffffffu, py[u], o);
                pz[u] = pz[u] + __shfl_xor_sync(0xffffffffu, pz[u], o);
            }
        }
#pragma unroll
        for (int w = 1; w < 8 / SUB; w <<= 1) {
#pragma unroll
            for (int u = 0; u + w < 8 / SUB; u += 2 * w) {
                px[u] = px[u] + px[u + w]; py[u] = py[u] + py[u + w]; pz[u] = pz[u] + pz[u + w];
            }
        }
        }
        ax = px[0]; ay = py[0]; az = pz[0];
        ax = sx + ax; ay = sy + ay; az = sz + az;
    }
    a[0] = ax; a[1] = ay; a[2] = az;
}

// Whole-grid regime, start of a group: publishes the bodies' starting positions, R_b and D_b, counts and fills the
// CTAs' lists (two scans of the group, tile by tile through shared memory: a lane scans for its body the partners
// j = sub, sub + SUB, .. (mod 8); a CTA reserves the chunks of its list with one atomic on a cursor -- where a list
// lies is irrelevant; within it the entries are in the order thread, residue class of j, ascending j).
// Two grid barriers; the positions go to buffer eval & 1 like a force evaluation's.
template <int ROWS, int SUB>
__device__ __forceinline__ void bs_build_lists(BsShared<ROWS>& S, const BsGlobal& Gm, int& eval, int i, int n, bool i_tp,
                                               int tp_mode, const double (&q)[3], const double (&v)[3],
                                               const double (&rci)[GENGA_BS_MAX_LEVELS], int nlevels, double dt, double mu,
                                               BsList<8 / SUB>& L)
{
    constexpr int NL = 8 / SUB;
    const int t = threadIdx.x, sub = t & (SUB - 1), lane = t & 31;
    const int p = eval & 1;
    eval++;
    const double x = q[0], y = q[1], z = q[2];
    const double rc0 = rci[0];
    const double bnd_i = bs_far_bound(rc0);
    const double lr_i = sqrt(bnd_i);
    const double la_i = i < n ? mu * (dt * dt) / (x * x + y * y + z * z) : 0.0;
    const double ld_i = sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]) * fabs(dt) + la_i;
    L.q0[0] = x; L.q0[1] = y; L.q0[2] = z;
    L.v0[0] = v[0]; L.v0[1] = v[1]; L.v0[2] = v[2];
    L.a2 = la_i * la_i;
    L.gmi = i < n ? fabs(__ldcg(Gm.gm + i)) : 0.0;               // (written by this body's first lane at the start of the group:
    L.gmi = __shfl_sync(0xffffffffu, L.gmi, (t & 31) & ~(SUB - 1));  //  the other lanes of the body take it from that lane)
    if (i < n && sub == 0) {
        Gm.x[p][i] = x; Gm.y[p][i] = y; Gm.z[p][i] = z;
        Gm.pk[p][2 * i] = make_double2(x, y); Gm.pk[p][2 * i + 1] = make_double2(z, L.gmi);
        Gm.vx[i] = v[0]; Gm.vy[i] = v[1]; Gm.vz[i] = v[2];
        Gm.lr[i] = lr_i; Gm.la[i] = la_i; Gm.ld[i] = ld_i;
    }
    if (Gm.tb == 0 && t == 0) *Gm.cursor = 0ULL;            // (its last readers passed several barriers ago)
    bs_gsync(S, Gm);
    L.cbase = 0; L.cchunks = 0;
    L.on = false;
    __shared__ int wtot[GENGA_BS_COOP_THREADS / 32];
    __shared__ long long cta_base;
    // FP32 copies of the staged tile for two conservative tests before the exact FP64 ones (which alone decide the
    // lists): of ~300 bodies within reach of a body's displacement bounds in the dense group of configs[3], ~80 pass the
    // FP32 closest-approach test, 77 are listed.  ftile = (x, y, z, h), h_b >= R_b + D_b + e_b, e_b >= the rounding of b's
    // coordinates to FP32: a pair can only pass the exact tests if |dq|_FP32 <= h_i + h_j (R = max(R_i, R_j) + D_i + D_j
    // <= h_i + h_j).  vtile = (v, A_b + e_b + f_b), f_b >= |dt| x the rounding of b's velocity; ltile = (R_b, f_b).
    // The FP32 closest approach is taken at the FP32 minimiser ts of |dq + dv tau|: the true distance there exceeds the
    // true minimum by at most |dv| |ts - tau*| <= sqrt(2 |dq| (f_i + f_j)) (the error of ts is that of dq.dv / dv.dv,
    // and |dv| |ts| <= |dv| |dt|), which is added to the radius with the e's and f's; 1.001 covers the FP32 roundings.
    __shared__ float4 ftile[ROWS];
    __shared__ float4 vtile[ROWS];
    __shared__ float2 ltile[ROWS];
    __shared__ double tvz[ROWS];                                 // the tile's velocities in FP64: S.rc[2], S.rc[3] and this
    const float fxi = (float)x, fyi = (float)y, fzi = (float)z, fvxi = (float)v[0], fvyi = (float)v[1], fvzi = (float)v[2];
    const float fdt = (float)dt;
    const float e_i = __fmul_ru(2.4e-7f, __fadd_ru(__fadd_ru(fabsf(fxi), fabsf(fyi)), fabsf(fzi)));
    const float f_i = __fmul_ru(__fmul_ru(2.4e-7f, __fadd_ru(__fadd_ru(fabsf(fvxi), fabsf(fvyi)), fabsf(fvzi))),
                                __fmul_ru(fabsf(fdt), 1.000001f));
    const float h_i = __fadd_ru(__fadd_ru(__double2float_ru(lr_i), __double2float_ru(ld_i)), e_i);
    const float lrf_i = __double2float_ru(lr_i), laf_i = __fadd_ru(__fadd_ru(__double2float_ru(la_i), e_i), f_i);
    const int cw = bs_chunk_words(nlevels);
    unsigned long long* const words = reinterpret_cast<unsigned long long*>(Gm.nbr);
    int cnt[NL];                                              // pass 0: entries of each of the lane's residue classes
    int lane_off = 0, ctotal = 0;                             // the lane's first entry within the CTA's list; its length
#pragma unroll
    for (int u = 0; u < NL; u++) cnt[u] = 0;
    for (int pass = 0; pass < 2; pass++) {                    // 0: count, 1: fill
        int c[NL];
#pragma unroll
        for (int u = 0; u < NL; u++) c[u] = 0;
        for (int j0 = 0; j0 < n; j0 += ROWS) {
            __syncthreads();
            if (t < ROWS && j0 + t < n) {
                S.x[t] = __ldcg(Gm.x[p] + j0 + t); S.y[t] = __ldcg(Gm.y[p] + j0 + t); S.z[t] = __ldcg(Gm.z[p] + j0 + t);
                S.gm[t] = __ldcg(Gm.gm + j0 + t);
                S.rcsq[t] = __ldcg(Gm.lr + j0 + t);
                S.rc[0][t] = __ldcg(Gm.ld + j0 + t);
                S.rc[1][t] = __ldcg(Gm.la + j0 + t);
                S.rc[2][t] = __ldcg(Gm.vx + j0 + t); S.rc[3][t] = __ldcg(Gm.vy + j0 + t); tvz[t] = __ldcg(Gm.vz + j0 + t);
                const float fxj = (float)S.x[t], fyj = (float)S.y[t], fzj = (float)S.z[t];
                const float fvxj = (float)S.rc[2][t], fvyj = (float)S.rc[3][t], fvzj = (float)tvz[t];
                const float e_j = __fmul_ru(2.4e-7f, __fadd_ru(__fadd_ru(fabsf(fxj), fabsf(fyj)), fabsf(fzj)));
                const float f_j = __fmul_ru(__fmul_ru(2.4e-7f, __fadd_ru(__fadd_ru(fabsf(fvxj), fabsf(fvyj)), fabsf(fvzj))),
                                            __fmul_ru(fabsf(fdt), 1.000001f));
                ftile[t] = make_float4(fxj, fyj, fzj,
                                       __fadd_ru(__fadd_ru(__double2float_ru(S.rcsq[t]), __double2float_ru(S.rc[0][t])), e_j));
                vtile[t] = make_float4(fvxj, fvyj, fvzj, __fadd_ru(__fadd_ru(__double2float_ru(S.rc[1][t]), e_j), f_j));
                ltile[t] = make_float2(__double2float_ru(S.rcsq[t]), f_j);
            }
            __syncthreads();
            if (i < n) {
                const int m = min(ROWS, n - j0);
                // First the FP32 test of the tile's bodies against this lane's, without a branch: one bit per body that
                // passes (a lane meets a candidate in 2 % of its tests, a WARP in half of them: taking the tests and the
                // follow-up of the hits in turn made every other test pay for a hit).  Then each lane's own hits.
                static_assert(ROWS <= 256, "one bit per j8 round of a tile");
                unsigned hits[NL];
#pragma unroll
                for (int u = 0; u < NL; u++) hits[u] = 0u;
#pragma unroll 4
                for (int j8 = 0; j8 < ROWS; j8 += 8) {
#pragma unroll
                    for (int u = 0; u < NL; u++) {
                        const int jj = j8 + sub + SUB * u;
                        const float4 fj = ftile[jj];                          // (beyond m: stale, masked below)
                        const float ex = fj.x - fxi, ey = fj.y - fyi, ez = fj.z - fzi, hh = __fadd_ru(fj.w, h_i);
                        const bool hit = jj < m && ex * ex + ey * ey + ez * ez <= __fmul_ru(__fmul_ru(hh, hh), 1.000002f);
                        hits[u] |= (hit ? 1u : 0u) << (j8 >> 3);
                    }
                }
#pragma unroll
                for (int u = 0; u < NL; u++) {
                    while (hits[u]) {
                        const int jj = 8 * (__ffs(hits[u]) - 1) + sub + SUB * u;
                        hits[u] &= hits[u] - 1u;
                        const float4 fj = ftile[jj];
                        const float ex = fj.x - fxi, ey = fj.y - fyi, ez = fj.z - fzi, hh = __fadd_ru(fj.w, h_i);
                        {
                            const float4 vj = vtile[jj];
                            const float2 lj = ltile[jj];
                            const float wxf = vj.x - fvxi, wyf = vj.y - fvyi, wzf = vj.z - fvzi;
                            const float w2f = wxf * wxf + wyf * wyf + wzf * wzf, dwf = ex * wxf + ey * wyf + ez * wzf;
                            float tsf = w2f > 0.0f ? __fdividef(-dwf, w2f) : 0.0f;
                            tsf = fdt > 0.0f ? fminf(fmaxf(tsf, 0.0f), fdt) : fmaxf(fminf(tsf, 0.0f), fdt);
                            const float cxf = ex + wxf * tsf, cyf = ey + wyf * tsf, czf = ez + wzf * tsf;
                            const float raf = __fadd_ru(__fadd_ru(fmaxf(lrf_i, lj.x), __fadd_ru(laf_i, vj.w)),
                                                        __fmul_ru(1.0001f, __fsqrt_ru(__fmul_ru(__fmul_ru(2.0f, hh), __fadd_ru(f_i, lj.y)))));
                            if (!(cxf * cxf + cyf * cyf + czf * czf <= __fmul_ru(__fmul_ru(raf, raf), 1.001f))) continue;
                        }
                        if (j0 + jj != i) {
                            const bool never = __double2hiint(S.gm[jj]) < 0 && (i_tp || tp_mode != 2);   // sec. 8.1
                            const double dx = S.x[jj] - x, dy = S.y[jj] - y, dz = S.z[jj] - z;
                            const double Rm = fmax(lr_i, S.rcsq[jj]);
                            const double R = Rm + (ld_i + S.rc[0][jj]);
                            // first the cheap test on the displacement bounds (implied by the one below), then the
                            // closest approach of the straight-line relative motion over [0, dt]
                            if (!never && dx * dx + dy * dy + dz * dz < R * R) {
                                const double wx = S.rc[2][jj] - v[0], wy = S.rc[3][jj] - v[1], wz = tvz[jj] - v[2];
                                const double w2 = wx * wx + wy * wy + wz * wz, dw = dx * wx + dy * wy + dz * wz;
                                double ts = w2 > 0.0 ? -dw / w2 : 0.0;            // unconstrained closest approach
                                ts = dt > 0.0 ? fmin(fmax(ts, 0.0), dt) : fmax(fmin(ts, 0.0), dt);
                                const double cx = dx + wx * ts, cy = dy + wy * ts, cz = dz + wz * ts;
                                const double Ra = Rm + (la_i + S.rc[1][jj]);
                                // (1 + 2^-30: the roundings of this test must not drop a pair the exact test keeps)
                                if (cx * cx + cy * cy + cz * cz < (Ra * Ra) * (1.0 + 9.313225746154785e-10)) {
                                    if (pass) {
                                        int e = lane_off + c[u];              // entry within the CTA's list
#pragma unroll
                                        for (int w = 0; w < NL; w++)
                                            if (w < u) e += cnt[w];
                                        const int jg = j0 + jj;
                                        unsigned long long* rec = words + (L.cbase + (e >> 5)) * cw + (e & 31);
                                        rec[0] = (unsigned long long)(unsigned)jg | ((unsigned long long)(unsigned)(t / SUB) << 32);
                                        rec[32] = (unsigned long long)__double_as_longlong(fmax(bnd_i, __ldcg(Gm.rcsq + jg)));
                                        for (int k = 0; k < nlevels; k++)
                                            rec[64 + 32 * k] = (unsigned long long)__double_as_longlong(
                                                1.0 / (0.9 * fmax(rci[k], __ldcg(Gm.rc[k] + jg))));
                                    }
                                    c[u]++;
                                }
                            }
                        }
                    }
                }
            }
        }
        if (pass) break;
        int total = 0;
#pragma unroll
        for (int u = 0; u < NL; u++) { cnt[u] = c[u]; total += c[u]; }
        int incl = total;                                         // inclusive scan over the CTA's threads
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int up = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += up;
        }
        __syncthreads();
        if (lane == 31) wtot[t >> 5] = incl;
        __syncthreads();
        int before = 0;
        ctotal = 0;
#pragma unroll
        for (int w = 0; w < GENGA_BS_COOP_THREADS / 32; w++) {
            if (w < (t >> 5)) before += wtot[w];
            ctotal += wtot[w];
        }
        lane_off = before + incl - total;
        const int chunks = (ctotal + 31) >> 5;
        if (t == 0) cta_base = chunks ? (long long)atomicAdd(Gm.cursor, (unsigned long long)chunks) : 0LL;
        bs_gsync(S, Gm);
        L.cbase = cta_base;
        L.cchunks = chunks;
        // team-uniform: all pairs instead if the lists do not fit
        if (__ldcg(Gm.cursor) * (unsigned long long)cw > (unsigned long long)(Gm.nbr_capacity / 2)) { L.cchunks = 0; return; }
    }
    // padding at the end of the CTA's last chunk: entries that belong to no body
    for (int e = ctotal + t; e < 32 * L.cchunks; e += GENGA_BS_COOP_THREADS)
        words[(L.cbase + (e >> 5)) * cw + (e & 31)] = 0xffffffffULL | (0x7fffULL << 32);
    L.on = true;
}

// maximum of e over the group (order-free); CTA- (and, COOP, grid-) uniform result
template <int MODE, int THREADS, int ROWS>
__device__ __forceinline__ double bs_group_max(BsShared<ROWS>& S, const BsGlobal& Gm, int& echeck, double e)
{
    constexpr bool COOP = MODE == GENGA_BS_MODE_COOP;
    const int t = threadIdx.x;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) e = fmax(e, __shfl_xor_sync(0xffffffffu, e, o));
    if (MODE == GENGA_BS_MODE_WARP) return e;                 // the group is the warp
    __syncthreads();
    if ((t & 31) == 0) S.red[t >> 5] = e;
    __syncthreads();
    if (t == 0) {
        double m = S.red[0];
#pragma unroll
        for (int w = 1; w < THREADS / 32; w++) m = fmax(m, S.red[w]);
        S.errmax = m;
    }
    __syncthreads();
    if (MODE == GENGA_BS_MODE_CLUSTER) {
        // each CTA publishes its maximum (two slots used in turn), one cluster barrier, everybody reads all of them
        cooperative_groups::cluster_group cl = cooperative_groups::this_cluster();
        const int slot = echeck & 1;
        echeck++;
        if (t == 0) S.emax[slot] = S.errmax;
        cl.sync();
        double m = 0.0;
#pragma unroll
        for (unsigned r = 0; r < GENGA_BS_CLUSTER; r++) m = fmax(m, *cl.map_shared_rank(&S.emax[slot], r));
        return m;
    }
    if (!COOP) return S.errmax;
    // non-negative doubles order like their bit patterns: atomicMax on the bits; four slots used in turn, the slot
    // two checks ahead is cleared after this check's barrier (its last readers passed the previous barrier)
    const int slot = echeck & 3;
    echeck++;
    if (t == 0) atomicMax(Gm.err + slot, (unsigned long long)__double_as_longlong(S.errmax));
    bs_gsync(S, Gm);
    const double m = __longlong_as_double((long long)__ldcg(Gm.err + slot));
    if (Gm.tb == 0 && t == 0) Gm.err[(slot + 2) & 3] = 0ULL;
    return m;
}

// Whole-grid regime: every CTA builds the same list of the next (up to GENGA_BS_BIG_LIST) groups with more than
// `small_max` bodies, in ascending order, scanning the offsets from group `scan_from` on, THREADS groups per round
// (a serial walk over tens of thousands of two-body groups cost 0.6 ms per call).  CTA-uniform results.
#define GENGA_BS_BIG_LIST 256
template <int THREADS>
__device__ __forceinline__ void bs_scan_large(const int* __restrict__ offsets, int n_groups, int small_max, int hi_max,
                                              int& scan_from, int* big, unsigned* wm, int& nbig)
{
    const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
    int count = 0;
    while (scan_from < n_groups && count + THREADS <= GENGA_BS_BIG_LIST) {
        const int g = scan_from + t;
        const int sz = g < n_groups ? offsets[g + 1] - offsets[g] : 0;
        const bool is_big = sz > small_max && (hi_max < 0 || sz <= hi_max);
        const unsigned m = __ballot_sync(0xffffffffu, is_big);
        __syncthreads();                                               // wm's previous readers are done
        if (lane == 0) wm[warp] = m;
        __syncthreads();
        int before = 0, total = 0;
#pragma unroll
        for (int w = 0; w < THREADS / 32; w++) {
            const int c = __popc(wm[w]);
            if (w < warp) before += c;
            total += c;
        }
        if (is_big) big[count + before + __popc(m & ((1u << lane) - 1u))] = g;
        count += total;
        scan_from += THREADS;
    }
    __syncthreads();
    nbig = count;
}

// WARP: warp w, w + (warps of the grid), ... integrates group w if it has at most 8 bodies.
// CTA : CTA g, g + gridDim.x, ... integrates group g if it has 9 .. 32 bodies.
// CLUSTER: cluster c, c + (clusters of the grid), ... of the groups with 33 .. 256 bodies (found by the same scan as below).
// COOP: the whole grid integrates, one after the other, the groups with more than `small_max` and at most `big_max`
//       bodies (two launches: a grid of one CTA per SM, whose barrier is cheap, for groups it can hold, and the full
//       co-resident grid for the rest); groups larger than the grid of a launch with big_max < 0 are reported and
//       left as they are.
template <int MODE, int THREADS, int SUB>
__device__ __forceinline__ void
bs_run(const double* __restrict__ pos_in, const double* __restrict__ vel_in, const double* __restrict__ mass,
          const double* __restrict__ rcrit, long long N, int nlevels, double G, double mu, double dt, double tol,
          const int* __restrict__ members, const int* __restrict__ offsets, const int* __restrict__ summary,
          double* __restrict__ pos, double* __restrict__ vel, int* __restrict__ status, const BsGlobal Gm_in, int small_max,
          long long n_massive, int tp_mode, int big_max, int vblock, int vgrid)
{
    BsGlobal Gm = Gm_in;
    // vblock / vgrid: this CTA's index and the number of CTAs of its regime (the warp and one-CTA regimes share a launch)
    constexpr bool COOP = MODE == GENGA_BS_MODE_COOP, WARP = MODE == GENGA_BS_MODE_WARP;
    constexpr bool CLUSTER = MODE == GENGA_BS_MODE_CLUSTER, LISTED = COOP || CLUSTER;
    constexpr int ROWS = COOP ? GENGA_BS_TILE : (WARP ? GENGA_BS_WARP_MAX : (MODE == GENGA_BS_MODE_CTA ? GENGA_BS_CTA_MAX : THREADS));
    constexpr int UNITS = WARP ? THREADS / 32 : 1;                      // groups in flight per CTA
    __shared__ BsShared<ROWS> Sall[UNITS];
    BsShared<ROWS>& S = Sall[WARP ? threadIdx.x >> 5 : 0];
    const int t = WARP ? (int)(threadIdx.x & 31) : (int)threadIdx.x;
    // this thread's body within the group (whole-grid regime: GENGA_BS_SUB consecutive lanes share a body and carry
    // identical copies of its state; they differ only in the part of the force sum they evaluate)
    // (cluster regime: the same, over the CTAs of the cluster: CTA r holds the bodies 32 r .. 32 r + 31)
    const int crank = CLUSTER ? (int)(blockIdx.x % GENGA_BS_CLUSTER) : 0;
    constexpr bool CTA = MODE == GENGA_BS_MODE_CTA;
    // whole-grid regime: this CTA's team (the whole grid, or team_ctas consecutive CTAs), and the team's slice of the scratch
    const int tctas = COOP ? (Gm.team_ctas ? Gm.team_ctas : (int)gridDim.x) : 1;
    const int team = COOP ? (int)blockIdx.x / tctas : 0, n_teams = COOP ? (int)gridDim.x / tctas : 1;
    if (COOP) {
        if (team >= n_teams) return;                                    // CTAs beyond the last whole team
        Gm.tb = (int)blockIdx.x - team * tctas;
        Gm.team_ctas = tctas;
        const long long off = (long long)team * tctas * THREADS / SUB;
#pragma unroll
        for (int h = 0; h < 2; h++) { Gm.x[h] += off; Gm.y[h] += off; Gm.z[h] += off; Gm.pk[h] += 2 * off; }
        Gm.sr += 3 * off;
        Gm.gm += off; Gm.rcsq += off; Gm.lr += off; Gm.la += off; Gm.ld += off; Gm.vx += off; Gm.vy += off; Gm.vz += off;
#pragma unroll
        for (int k = 0; k < GENGA_BS_MAX_LEVELS; k++) Gm.rc[k] += off;
        Gm.err += 16 * team; Gm.cursor = Gm.err + 4; Gm.bar = Gm.err + 5;
        Gm.nbr_capacity = (Gm.nbr_capacity / n_teams) & ~3LL;     // (a team's slice starts on a 16-byte boundary)
        Gm.nbr += (long long)team * Gm.nbr_capacity;
        if (threadIdx.x == 0) S.bar_target = 0ULL;
    }
    // (whole-grid regime: the group's bodies are dealt round the team's CTAs, body i to CTA i mod tctas: every CTA of the
    // team gets its share whatever the group's size)
    const int i = COOP ? (t / SUB) * tctas + Gm.tb : (CLUSTER ? (crank * THREADS + t) / SUB : (CTA ? t / SUB : t));
    const bool writer = WARP || (t & (SUB - 1)) == 0;
    const long long capacity = COOP ? (long long)tctas * THREADS / SUB : ROWS;
    const int n_groups = summary[0];
    int eval = 0, echeck = 0;
    const int g0 = COOP ? 0 : (WARP ? (int)(vblock * UNITS + (threadIdx.x >> 5)) : vblock);
    const int gstep = COOP ? 1 : vgrid * UNITS;
    __shared__ int big[LISTED ? GENGA_BS_BIG_LIST : 1];
    __shared__ unsigned wm[THREADS / 32];
    // whole-grid regime: every CTA walks the whole list; cluster regime: cluster c takes the entries c, c + clusters, ..
    const int lfirst = CLUSTER ? (int)(blockIdx.x / GENGA_BS_CLUSTER) : team;
    const int lstep = CLUSTER ? (int)(gridDim.x / GENGA_BS_CLUSTER) : n_teams;
    int scan_from = 0, nbig = 0, ib = 0;
    if (LISTED && summary[2] <= small_max) return;                      // no group for this regime (grid-uniform)
    for (int g = g0;; g += gstep) {
        if (LISTED) {
            while (ib >= nbig && scan_from < n_groups) {
                ib = ib - nbig + (nbig == 0 && scan_from == 0 ? lfirst : 0);      // position within the next batch
                bs_scan_large<THREADS>(offsets, n_groups, small_max, CLUSTER ? THREADS : big_max, scan_from, big, wm, nbig);
            }
            if (ib >= nbig) break;
            g = big[ib];
            ib += lstep;
        } else if (g >= n_groups) break;
        const int first = offsets[g], n = offsets[g + 1] - first;
        // the other regimes' groups (grid- / CTA- / warp-uniform)
        if (COOP ? (n <= small_max || (big_max >= 0 && n > big_max))
                 : (WARP ? n > GENGA_BS_SEQ_MAX : (CTA ? (n <= GENGA_BS_SEQ_MAX || n > GENGA_BS_CTA_MAX) : false))) continue;
        // (listed regimes: the scan has already applied these bounds)
        if (n > capacity) {
            if (t == 0 && (COOP ? Gm.tb == 0 : blockIdx.x == 0)) atomicOr(status, GENGA_STATUS_GROUP_TOO_LARGE);
            continue;
        }
        const bool active = i < n;
        const long long b = active ? members[first + i] : 0;
        const bool i_tp = b >= n_massive;
        double q[3] = {0.0, 0.0, 0.0}, v[3] = {0.0, 0.0, 0.0}, rci[GENGA_BS_MAX_LEVELS] = {0.0, 0.0, 0.0, 0.0};
        if (!COOP) bs_sync<MODE>();                                     // the previous group's readers are done
        if (active) {
#pragma unroll
            for (int c = 0; c < 3; c++) { q[c] = pos_in[c * N + b]; v[c] = vel_in[c * N + b]; }
            // semi-active particles (b >= n_massive; n_massive = N in TP 0) carry the sign bit: see GENGA_BS_PAIR
            const double gm = b >= n_massive ? -(G * mass[b]) : G * mass[b];
            for (int k = 0; k < nlevels; k++) rci[k] = rcrit[(long long)k * N + b];
            if (COOP) {
                if (writer) {
                    Gm.gm[i] = gm;
                    Gm.sr[3 * i] = make_double2(gm, rci[0]); Gm.sr[3 * i + 1] = make_double2(rci[1], rci[2]);
                    Gm.sr[3 * i + 2] = make_double2(rci[3], 0.0);
                    Gm.rcsq[i] = bs_far_bound(rci[0]);
                    for (int k = 0; k < nlevels; k++) Gm.rc[k][i] = rci[k];
                }
            } else if (WARP) {
                S.gm[i] = gm;
                S.rcsq[i] = bs_far_bound(rci[0]);
                for (int k = 0; k < nlevels; k++) S.rc[k][i] = rci[k];
            }
        }
        if (CLUSTER || CTA) {                                           // every CTA stages the whole group's G m and radii
            for (int idx = t; idx < n; idx += THREADS) {
                const long long bj = members[first + idx];
                S.gm[idx] = bj >= n_massive ? -(G * mass[bj]) : G * mass[bj];
                S.rcsq[idx] = bs_far_bound(rcrit[bj]);
                for (int k = 0; k < nlevels; k++) S.rc[k][idx] = rcrit[(long long)k * N + bj];
            }
        }
        // (COOP: G m and the radii are read by other CTAs only after the first force evaluation's grid barrier;
        //  the previous group's last readers passed a grid barrier -- its last error check -- before anyone gets here)
        BsList<8 / SUB> L;
        L.on = false;
        if (COOP) bs_build_lists<ROWS, SUB>(S, Gm, eval, i, n, i_tp, tp_mode, q, v, rci, nlevels, dt, mu, L);
        double Pq[GENGA_BS_KMAX][3], Pv[GENGA_BS_KMAX][3];             // P[j] = T_{k-1,j} of the extrapolation tableau
        double a0[3], cq[3], cv[3], dq[3], dv[3];
        double done = 0.0, H = dt;
        bool fail = false;
        int n_acc = 0, n_rej = 0, n_fev = 0;                           // group-uniform, like every decision below
        while (done != dt) {                                           // all decisions below are group-uniform
            if ((dt > 0.0 && done + H > dt) || (dt < 0.0 && done + H < dt)) H = dt - done;
            bs_force<MODE, ROWS, SUB>(S, Gm, eval, i, n, nlevels, i_tp, tp_mode, mu, rci, q, a0, L, done, status);
            n_fev++;
            int halvings = 0, kconv = 0;
            for (;;) {
                bool ok = false;
                for (int k = 0; k < GENGA_BS_KMAX; k++) {
                    const int nk = 2 * (k + 1);
                    n_fev += nk;
                    {   // modified midpoint over H with nk sub-steps: (q, v) -> (cq, cv) = T_{k,0}
                        const double h = H / (double)nk, h2 = 2.0 * h;
                        double qm[3], vm[3], qn[3], vn[3], a[3];
#pragma unroll
                        for (int c = 0; c < 3; c++) { qm[c] = q[c]; vm[c] = v[c]; qn[c] = q[c] + h * v[c]; vn[c] = v[c] + h * a0[c]; }
                        for (int m = 1; m < nk; m++) {
                            bs_force<MODE, ROWS, SUB>(S, Gm, eval, i, n, nlevels, i_tp, tp_mode, mu, rci, qn, a, L,
                                                      done + (double)m * h, status);
#pragma unroll
                            for (int c = 0; c < 3; c++) {
                                const double qs = qm[c] + h2 * vn[c], vs = vm[c] + h2 * a[c];
                                qm[c] = qn[c]; vm[c] = vn[c]; qn[c] = qs; vn[c] = vs;
                            }
                        }
                        bs_force<MODE, ROWS, SUB>(S, Gm, eval, i, n, nlevels, i_tp, tp_mode, mu, rci, qn, a, L, done + H, status);
#pragma unroll
                        for (int c = 0; c < 3; c++) {
                            cq[c] = 0.5 * (qn[c] + qm[c] + h * vn[c]);
                            cv[c] = 0.5 * (vn[c] + vm[c] + h * a[c]);
                        }
                    }
                    for (int j = 1; j <= k; j++) {
                        const double ratio = (double)nk / (double)(2 * (k - j + 1));      // n_k / n_{k-j}
                        const double den = ratio * ratio - 1.0;
#pragma unroll
                        for (int c = 0; c < 3; c++) {
                            const double lq = cq[c], lv = cv[c];                          // T_{k,j-1}
                            const double nq = lq + (lq - Pq[j - 1][c]) / den;             // T_{k,j}
                            const double nv = lv + (lv - Pv[j - 1][c]) / den;
                            Pq[j - 1][c] = lq; Pv[j - 1][c] = lv;
                            cq[c] = nq; cv[c] = nv;
                            dq[c] = nq - lq; dv[c] = nv - lv;                             // after j = k: T_kk - T_k,k-1
                        }
                    }
#pragma unroll
                    for (int c = 0; c < 3; c++) { Pq[k][c] = cq[c]; Pv[k][c] = cv[c]; }   // T_kk
                    if (k > 0) {
                        double e = 0.0;
                        if (active) {
                            double eq2 = 0.0, sq2 = 0.0, ev2 = 0.0, sv2 = 0.0;
#pragma unroll
                            for (int c = 0; c < 3; c++) {
                                eq2 = eq2 + dq[c] * dq[c]; sq2 = sq2 + cq[c] * cq[c];
                                ev2 = ev2 + dv[c] * dv[c]; sv2 = sv2 + cv[c] * cv[c];
                            }
                            e = fmax(sqrt(eq2) / sqrt(sq2), sqrt(ev2) / sqrt(sv2));
                        }
                        if (bs_group_max<MODE, THREADS, ROWS>(S, Gm, echeck, e) <= tol) { ok = true; kconv = k + 1; break; }
                    }
                }
                if (ok) break;
                n_rej++;
                if (++halvings > GENGA_BS_MAX_HALVINGS) { fail = true; break; }
                H = 0.5 * H;
            }
            if (fail) break;
            n_acc++;
#pragma unroll
            for (int c = 0; c < 3; c++) { q[c] = cq[c]; v[c] = cv[c]; }
            if ((dt > 0.0 && done + H >= dt) || (dt < 0.0 && done + H <= dt)) done = dt;
            else done = done + H;
            if (kconv <= 5) H = 2.0 * H;
        }
        if (fail && t == 0 && (!COOP || Gm.tb == 0)) atomicOr(status, GENGA_STATUS_BS_NOT_CONVERGED);
        if (active && writer) {                                        // (after a failure: the state at the last accepted time)
#pragma unroll
            for (int c = 0; c < 3; c++) { pos[c * N + b] = q[c]; vel[c * N + b] = v[c]; }
            if (i == 0) {                                              // one thread per group: the step-size control's record
                atomicAdd(Gm.totals + 0, (unsigned long long)n_acc); atomicAdd(Gm.totals + 1, (unsigned long long)n_rej);
                atomicAdd(Gm.totals + 2, (unsigned long long)n_fev); atomicAdd(Gm.totals + 3, 1ULL);
                if (Gm.stats && g < Gm.stats_rows) Gm.stats[g] = make_int4(n_acc, n_rej, n_fev, n);
            }
        }
    }
    // no CTA of a cluster leaves while another may still read its shared memory
    if (CLUSTER) cooperative_groups::this_cluster().sync();
}

#define GENGA_BS_ARGS                                                                                                   \
    const double *__restrict__ pos_in, const double *__restrict__ vel_in, const double *__restrict__ mass,              \
        const double *__restrict__ rcrit, long long N, int nlevels, double G, double mu, double dt, double tol,         \
        const int *__restrict__ members, const int *__restrict__ offsets, const int *__restrict__ summary,              \
        double *__restrict__ pos, double *__restrict__ vel, int *__restrict__ status, const BsGlobal Gm, int small_max, \
        long long n_massive, int tp_mode, int big_max
#define GENGA_BS_PASS                                                                                                    \
    pos_in, vel_in, mass, rcrit, N, nlevels, G, mu, dt, tol, members, offsets, summary, pos, vel, status, Gm, small_max, \
        n_massive, tp_mode, big_max

template <int MODE, int THREADS, int SUB = 1>
// (8 CTAs of 64 threads per SM whatever the variant: the capacities of the whole-grid regime -- 9472 bodies at eight
// lanes each on 148 SMs, twice that at four, .. -- must not move with the register allocator's mood)
__global__ void __launch_bounds__(THREADS, 512 / THREADS) bs_kernel(GENGA_BS_ARGS)
{
    bs_run<MODE, THREADS, SUB>(GENGA_BS_PASS, (int)blockIdx.x, (int)gridDim.x);
}

// the warp regime (CTAs below `split`) and the one-CTA regime (the rest) in ONE launch: their groups are independent, and
// a launch of its own for the few 9 .. 32-body groups would only add their duration to the step
__global__ void __launch_bounds__(GENGA_BS_THREADS) bs_small_kernel(GENGA_BS_ARGS, int split)
{
    if ((int)blockIdx.x < split)
        bs_run<GENGA_BS_MODE_WARP, GENGA_BS_THREADS, 1>(GENGA_BS_PASS, (int)blockIdx.x, split);
    else
        bs_run<GENGA_BS_MODE_CTA, GENGA_BS_THREADS, GENGA_BS_SUB>(GENGA_BS_PASS, (int)blockIdx.x - split,
                                                                  (int)gridDim.x - split);
}

// the cluster regime: GENGA_BS_CLUSTER CTAs per cluster (the grid is a multiple of it)
__global__ void __cluster_dims__(GENGA_BS_CLUSTER, 1, 1) __launch_bounds__(GENGA_BS_THREADS) bs_cluster_kernel(GENGA_BS_ARGS)
{
    bs_run<GENGA_BS_MODE_CLUSTER, GENGA_BS_THREADS, GENGA_BS_SUB>(GENGA_BS_PASS, (int)blockIdx.x, (int)gridDim.x);
}

}  // namespace genga
