// kick_sym_kernel: the level-0 pair loop over the massive bodies with every UNORDERED pair evaluated once
// (eq. 3 PAPER.md:63-64 is symmetric in i and j: the force on i and the reaction on j come from one r^-3).
//
// Why: an ordered pair costs 16 FP64-pipe instructions, an unordered pair 20 (3 DADD + 3 for r^2 + 6 for r^-3 + 2
// products with G m_j, G m_i + 6 accumulating DFMAs) instead of 32 -- measured 46.7 issue cycles per warp and unordered
// pair against 2 x 36 (profiles/ncu_r02*.md).  The FP64 pipe's dispatch port is the bottleneck (2 cycles per FP64
// instruction, 1 per anything else), so the loop is built to issue as little else as possible: 6 i-bodies per thread.
//
// How.  The pair matrix of the massive records is cut into rows (i-blocks of 1536 records) x j-tiles of 256 records;
// row I only holds the tiles jt >= 6 I (genga_kick_variants.h).  The 6 tiles that overlap the i-block itself (DIAGONAL)
// are evaluated one-sidedly exactly as kick_kernel does.  In every other tile (SYMMETRIC) a warp walks the tile's
// eight 32-record groups; lane l starts a group at its record l and moves on by one record per step (32 steps):
// at step s it evaluates its 6 i-bodies against j-record (l + s) mod 32, read from shared memory (every lane another
// record: conflict-free), adds s_i d to its own sums and -s_j d to the j-record's running reaction sum, which travels
// round the warp by shuffle (3 doubles per step) and is back at lane l after 32 steps.  The eight warps of the CTA
// visit the groups in rotated order (warp w starts at group w), and hand a group's reaction sum on through shared
// memory in a fixed order (a sequence counter per group: warp g, g-1, ..., g-7 mod 8), so the sum of a tile is a
// fixed function of the inputs; the last warp writes it to the tile's slot of the reaction scratch
// and reduce_kernel adds the slots of a record in ascending row order.
//
// Filter, culling and the candidate list are those of kick_kernel; a pair of a symmetric tile that trips the filter
// (now the exact per-pair rule hi(r^2) < max(fw_i, fw_j)) contributes exactly 0 to BOTH sides and is queued ONCE as a
// symmetric candidate (~i-record, j-record): exact_kernel adds both forces and does the pair's bookkeeping.
//
// No code, header, table or helper is shared with oracle/.
#pragma once
#include "genga_kick_kernels.cuh"

namespace genga {

// one unordered pair: i += s_i d, j -= s_j d.  20 FP64-pipe instructions.
__device__ __forceinline__ void pair_sym_bare(double xj, double yj, double zj, double gmj,
                                              double xi, double yi, double zi, double gmi,
                                              double& ax, double& ay, double& az, double& rx, double& ry, double& rz)
{
    const double dx = __dsub_rn(xj, xi), dy = __dsub_rn(yj, yi), dz = __dsub_rn(zj, zi);
    const double r2 = fma(dz, dz, fma(dy, dy, __dmul_rn(dx, dx)));
    double y0;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y0) : "d"(r2));
    const double t = __dmul_rn(y0, y0);
    const double e = fma(-r2, t, 1.0);
    const double u = __dmul_rn(t, y0);
    const double c = fma(1.875, e, 1.5);
    const double q = fma(e, c, 1.0);
    const double w = __dmul_rn(u, q);                       // r^-3
    const double si = __dmul_rn(gmj, w), sj = __dmul_rn(gmi, w);
    ax = fma(si, dx, ax); ay = fma(si, dy, ay); az = fma(si, dz, az);
    rx = fma(-sj, dx, rx); ry = fma(-sj, dy, ry); rz = fma(-sj, dz, rz);
}

// the same with the filter: a tripped pair adds exactly 0 to both sides
__device__ __forceinline__ bool pair_sym_fast(double xj, double yj, double zj, double gmj,
                                              double xi, double yi, double zi, double gmi, int thr,
                                              double& ax, double& ay, double& az, double& rx, double& ry, double& rz)
{
    const double dx = __dsub_rn(xj, xi), dy = __dsub_rn(yj, yi), dz = __dsub_rn(zj, zi);
    const double r2 = fma(dz, dz, fma(dy, dy, __dmul_rn(dx, dx)));
    const bool trig = __double2hiint(r2) < thr;
    const double y0 = rsqrt_seed_unless(r2, trig);
    const double t = __dmul_rn(y0, y0);
    const double e = fma(-r2, t, 1.0);
    const double u = __dmul_rn(t, y0);
    const double c = fma(1.875, e, 1.5);
    const double q = fma(e, c, 1.0);
    const double w = __dmul_rn(u, q);
    const double si = __dmul_rn(gmj, w), sj = __dmul_rn(gmi, w);
    ax = fma(si, dx, ax); ay = fma(si, dy, ay); az = fma(si, dz, az);
    rx = fma(-sj, dx, rx); ry = fma(-sj, dy, ry); rz = fma(-sj, dz, rz);
    return trig;
}

// acquire / release on a shared-memory word (the hand-over counters of the reaction sums)
__device__ __forceinline__ int ld_acquire_shared(const volatile int* q)
{
    int v;
    asm volatile("ld.acquire.cta.shared.s32 %0, [%1];" : "=r"(v) : "r"(smem_u32(const_cast<const int*>(q))) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_shared(volatile int* q, int v)
{
    asm volatile("st.release.cta.shared.s32 [%0], %1;" ::"r"(smem_u32(const_cast<int*>(q))), "r"(v) : "memory");
}

template <int JT>
struct alignas(128) SymStage {
    double2 xy[JT];
    double2 zm[JT];
    float4 blo[JT / GENGA_GROUP];
    float4 bhi[JT / GENGA_GROUP];
    int fw[JT];
};

struct SymParams {
    int n_rows;                        // i-blocks
    int r;                             // tiles_per_iblock
    double* __restrict__ react;        // [n_tiles][3][JT]
    const long long* __restrict__ cta_t0;   // [n_ctas + 1] first tile of every CTA (genga_kick_plan_sym_table)
};

template <int THREADS, int IPT, int STAGES>
__global__ void __launch_bounds__(THREADS, 1) kick_sym_kernel(const KickParams p, const SymParams sp)
{
    constexpr int WARPS = THREADS / 32;
    constexpr int JT = 32 * WARPS;                          // one group per warp and phase
    constexpr int IB = THREADS * IPT;
    constexpr int NG = JT / GENGA_GROUP;
    constexpr uint32_t TILE_BYTES = JT * 32 + NG * 32 + JT * 4;
    static_assert(NG == WARPS && NG <= 32, "one j-group per warp and phase");
    static_assert(4 * IPT <= 32, "one trigger bit per pair of four steps");
    __shared__ SymStage<JT> st[STAGES];
    __shared__ __align__(8) uint64_t full[STAGES];
    __shared__ __align__(8) uint64_t empty[STAGES];
    __shared__ double rs[3][JT];                            // a group's reaction sum on its way through the warps
    __shared__ volatile int cnt[NG];                        // contributions a group's sum has taken so far
    __shared__ float4 wblo[WARPS], wbhi[WARPS];             // box of each warp's i-records (.w of lo: largest filter word)
    __shared__ float4 wslo[WARPS][IPT], wshi[WARPS][IPT];   // ... and of each of its IPT slices of 32 records
    __shared__ CandCursor ccs[WARPS];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int woff = warp * (32 * IPT) + lane;
    const long long t0 = sp.cta_t0[blockIdx.x], t1 = sp.cta_t0[blockIdx.x + 1];
    if (t0 >= t1) return;

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < STAGES; s++) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], WARPS);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (tid < NG) cnt[tid] = 0;
    if (lane == 0) { ccs[warp].base = 0; ccs[warp].fill = GENGA_CAND_BLOCK; ccs[warp].over = false; }
    __syncthreads();

    // (row, jt) of the tiles t0, t0 + 1, ...: one cursor for the producer (thread 0), one for the consumers
    const int first_row = sym_row_of(t0, p.n_j_tiles, sp.r, sp.n_rows);
    const int first_jt = first_row * sp.r + (int)(t0 - sym_row_begin(first_row, p.n_j_tiles, sp.r));
    auto advance = [&](int& row, int& jt) {
        if (++jt == p.n_j_tiles) { ++row; jt = row * sp.r; }
    };
    int prow = first_row, pjt = first_jt;
    auto issue = [&](int g) {                               // thread 0 only, g = 0, 1, 2, ... in this order
        const int s = g % STAGES;
        if (g >= STAGES) mbar_wait(&empty[s], (uint32_t)((g / STAGES - 1) & 1));
        mbar_expect_tx(&full[s], TILE_BYTES);
        const size_t j0 = (size_t)pjt * JT;                 // a multiple of 256: every offset 16-byte aligned
        bulk_g2s(st[s].xy, p.rxy + j0, JT * 16, &full[s]);
        bulk_g2s(st[s].zm, p.rzm + j0, JT * 16, &full[s]);
        bulk_g2s(st[s].blo, p.cblo + j0 / GENGA_GROUP, NG * 16, &full[s]);
        bulk_g2s(st[s].bhi, p.cbhi + j0 / GENGA_GROUP, NG * 16, &full[s]);
        bulk_g2s(st[s].fw, p.rfw + j0, JT * 4, &full[s]);
        advance(prow, pjt);
    };
    const int n_it = (int)(t1 - t0);
    if (tid == 0)
        for (int g = 0; g < STAGES && g < n_it; g++) issue(g);

    double xi[IPT], yi[IPT], zi[IPT], gi[IPT], ax[IPT], ay[IPT], az[IPT];
    int row = first_row, jt = first_jt, cur_row = -1;
    int n_sym = 0;                                          // symmetric tiles done: numbers the hand-over of the reaction sums

    auto flush = [&]() {
        const size_t base = ((size_t)blockIdx.x * p.max_segs + (cur_row - first_row)) * 3 * IB;
#pragma unroll
        for (int k = 0; k < IPT; k++) {
            const int off = woff + k * 32;
            p.partial[base + off] = ax[k];
            p.partial[base + IB + off] = ay[k];
            p.partial[base + 2 * IB + off] = az[k];
        }
    };
    // the filter words of the thread's i-records, fetched only where a group needs the checked loop
    auto load_fi = [&](int (&fi)[IPT]) {
#pragma unroll
        for (int k = 0; k < IPT; k++) {
            const size_t r = (size_t)cur_row * IB + woff + k * 32;
            fi[k] = r < (size_t)p.i_rec_end ? __ldg(p.rfw + r) : -1;
        }
    };

    for (int it = 0; it < n_it; ++it) {
        const int s = it % STAGES;
        if (row != cur_row) {
            if (cur_row >= 0) flush();
            cur_row = row;
            float4 lo = make_float4(3.0e38f, 3.0e38f, 3.0e38f, 0.0f), hi = make_float4(-3.0e38f, -3.0e38f, -3.0e38f, 0.0f);
            int wfw = -1;
#pragma unroll
            for (int k = 0; k < IPT; k++) {
                const size_t r = (size_t)row * IB + woff + k * 32;
                ax[k] = ay[k] = az[k] = 0.0;
                if (r >= (size_t)p.i_rec_end) {             // whole groups of 32 records (i_rec_end is a multiple of 32)
                    xi[k] = yi[k] = zi[k] = GENGA_SENTINEL_POS;
                    gi[k] = 0.0;
                    if (lane == 0) {                        // an empty box, near to nothing
                        wslo[warp][k] = make_float4(3.0e38f, 3.0e38f, 3.0e38f, __int_as_float(-1));
                        wshi[warp][k] = make_float4(-3.0e38f, -3.0e38f, -3.0e38f, 0.0f);
                    }
                    continue;
                }
                const double2 a = p.rxy[r], b = p.rzm[r];
                xi[k] = a.x; yi[k] = a.y; zi[k] = b.x; gi[k] = b.y;
                const float4 glo = p.cblo[r / GENGA_GROUP], ghi = p.cbhi[r / GENGA_GROUP];
                if (lane == 0) { wslo[warp][k] = glo; wshi[warp][k] = ghi; }
                lo.x = fminf(lo.x, glo.x); lo.y = fminf(lo.y, glo.y); lo.z = fminf(lo.z, glo.z);
                hi.x = fmaxf(hi.x, ghi.x); hi.y = fmaxf(hi.y, ghi.y); hi.z = fmaxf(hi.z, ghi.z);
                wfw = max(wfw, __float_as_int(glo.w));
            }
            __syncwarp();                                   // the previous row's readers of the warp's box are done
            if (lane == 0) { lo.w = __int_as_float(wfw); wblo[warp] = lo; wbhi[warp] = hi; }
            __syncwarp();
        }
        mbar_wait(&full[s], (uint32_t)((it / STAGES) & 1));
        const SymStage<JT>& S = st[s];
        unsigned nearmask;
        {
            const float4 lo = wblo[warp], hi = wbhi[warp];
            const bool mine_near = lane < NG ? boxes_near(lo, hi, __float_as_int(lo.w), S.blo[lane], S.bhi[lane]) : false;
            nearmask = __ballot_sync(0xffffffffu, mine_near);
        }
        const bool diag = jt < (row + 1) * sp.r;            // the tile overlaps the i-block: one-sided, as kick_kernel

        if (diag) {
#pragma unroll 1
            for (int g = 0; g < NG; g++) {
                const int j0 = g * GENGA_GROUP;
                if (!((nearmask >> g) & 1u)) {
#pragma unroll 2
                    for (int u = 0; u < GENGA_GROUP; u++) {
                        const double2 xy = S.xy[j0 + u], zm = S.zm[j0 + u];
#pragma unroll
                        for (int k = 0; k < IPT; k++)
                            pair_bare(xy.x, xy.y, zm.x, zm.y, xi[k], yi[k], zi[k], ax[k], ay[k], az[k]);
                    }
                    continue;
                }
                int fi[IPT];
                load_fi(fi);
                CandCursor cc = ccs[warp];
#pragma unroll 1
                for (int jj = j0; jj < j0 + GENGA_GROUP; jj += 4) {
                    unsigned tm = 0;                        // bit u * IPT + k: pair (k, jj + u) tripped the filter
#pragma unroll
                    for (int u = 0; u < 4; u++) {
                        const double2 xy = S.xy[jj + u], zm = S.zm[jj + u];
                        const int fj = S.fw[jj + u];
#pragma unroll
                        for (int k = 0; k < IPT; k++) {
                            bool trig = false;
                            pair_fast(xy.x, xy.y, zm.x, zm.y, xi[k], yi[k], zi[k], max(fi[k], fj), ax[k], ay[k], az[k], trig);
                            tm |= (trig ? 1u : 0u) << (u * IPT + k);
                        }
                    }
                    unsigned todo = __reduce_or_sync(0xffffffffu, tm);
                    while (todo) {                          // warp-uniform: the (u, k) some lane tripped
                        const int b = __ffs(todo) - 1;
                        todo &= todo - 1;
                        push_candidates(p, cc, (tm >> b) & 1u, row * IB + woff + (b % IPT) * 32, jt * JT + jj + b / IPT);
                    }
                }
                __syncwarp();
                if (lane == 0) ccs[warp] = cc;
                __syncwarp();
            }
        } else {
            const int src = (lane + 1) & 31;
#pragma unroll 1
            for (int ph = 0; ph < WARPS; ph++) {
                const int g = (warp + ph) % NG, j0 = g * GENGA_GROUP;
                double rx = 0.0, ry = 0.0, rz = 0.0;
                // the warp's box (256 records) is near the group: look again slice by slice (32 records each)
                bool checked = (nearmask >> g) & 1u;
                if (checked) {
                    const bool kn = lane < IPT ? boxes_near(wslo[warp][lane], wshi[warp][lane], __float_as_int(wslo[warp][lane].w),
                                                            S.blo[g], S.bhi[g]) : false;
                    checked = __ballot_sync(0xffffffffu, kn) != 0u;
                }
                if (!checked) {
#pragma unroll 2
                    for (int q = 0; q < 32; q++) {
                        const int jj = j0 + ((lane + q) & 31);
                        const double2 xy = S.xy[jj], zm = S.zm[jj];
#pragma unroll
                        for (int k = 0; k < IPT; k++)
                            pair_sym_bare(xy.x, xy.y, zm.x, zm.y, xi[k], yi[k], zi[k], gi[k], ax[k], ay[k], az[k], rx, ry, rz);
                        rx = __shfl_sync(0xffffffffu, rx, src);
                        ry = __shfl_sync(0xffffffffu, ry, src);
                        rz = __shfl_sync(0xffffffffu, rz, src);
                    }
                } else {
                    int fi[IPT];
                    load_fi(fi);
                    CandCursor cc = ccs[warp];
#pragma unroll 1
                    for (int q0 = 0; q0 < 32; q0 += 4) {
                        unsigned tm = 0;                    // bit u * IPT + k: pair (k, record of step q0 + u) tripped the filter
#pragma unroll
                        for (int u = 0; u < 4; u++) {
                            const int jj = j0 + ((lane + q0 + u) & 31);
                            const double2 xy = S.xy[jj], zm = S.zm[jj];
                            const int fj = S.fw[jj];
#pragma unroll
                            for (int k = 0; k < IPT; k++) {
                                const bool trig = pair_sym_fast(xy.x, xy.y, zm.x, zm.y, xi[k], yi[k], zi[k], gi[k],
                                                                max(fi[k], fj), ax[k], ay[k], az[k], rx, ry, rz);
                                tm |= (trig ? 1u : 0u) << (u * IPT + k);
                            }
                            rx = __shfl_sync(0xffffffffu, rx, src);
                            ry = __shfl_sync(0xffffffffu, ry, src);
                            rz = __shfl_sync(0xffffffffu, rz, src);
                        }
                        unsigned todo = __reduce_or_sync(0xffffffffu, tm);
                        while (todo) {                      // warp-uniform: the (u, k) some lane tripped
                            const int b = __ffs(todo) - 1;
                            todo &= todo - 1;
                            const int jrec = jt * JT + j0 + ((lane + q0 + b / IPT) & 31);
                            // queued once, as a symmetric candidate: exact_kernel serves both bodies
                            push_candidates(p, cc, (tm >> b) & 1u, ~(row * IB + woff + (b % IPT) * 32), jrec);
                        }
                    }
                    __syncwarp();
                    if (lane == 0) ccs[warp] = cc;
                    __syncwarp();
                }
                // The group's reaction sum goes from warp to warp in a fixed order: this is contribution `ph` of the
                // CTA's symmetric tile number n_sym.  (rx now belongs to record j0 + lane again.)
                // (every lane polls the same word: the decision is warp-uniform and the warp stays converged -- a spin
                // by one lane left the warp split, every instruction of the pair loop issued twice)
                const int seq = n_sym * WARPS + ph;
                while (ld_acquire_shared(&cnt[g]) != seq) { }
                __syncwarp();
                if (ph > 0) {
                    rx = __dadd_rn(rs[0][j0 + lane], rx); ry = __dadd_rn(rs[1][j0 + lane], ry); rz = __dadd_rn(rs[2][j0 + lane], rz);
                }
                if (ph < WARPS - 1) {
                    rs[0][j0 + lane] = rx; rs[1][j0 + lane] = ry; rs[2][j0 + lane] = rz;
                } else {
                    double* o = sp.react + (size_t)(t0 + it) * (3 * JT) + j0 + lane;
                    o[0] = rx; o[JT] = ry; o[2 * JT] = rz;
                }
                __syncwarp();
                if (lane == 0) st_release_shared(&cnt[g], seq + 1);
                __syncwarp();
            }
            n_sym++;
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[s]);              // this warp is done with stage s
        if (tid == 0 && it >= 1 && it - 1 + STAGES < n_it) issue(it - 1 + STAGES);
        advance(row, jt);
    }
    flush();
    {
        CandCursor cc = ccs[warp];
        if (cc.fill < GENGA_CAND_BLOCK) close_block(p, cc);
    }
}

}  // namespace genga
