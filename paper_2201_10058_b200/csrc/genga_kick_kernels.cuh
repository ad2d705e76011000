// sm_100a kernels of the GENGA kick + close-encounter pre-check.
//
//   pack_kernel    O(N): writes the body RECORDS the pair loop reads (positions, G m, filter word,
//                  caller's index) in the library's internal order, the per-chunk filter maxima,
//                  and clears the encounter counters.
//   kick_kernel    O(N * n_massive): the pair loop (eq. 3 PAPER.md:63-64 with the weights of
//                  eq. 62-63, fused with the pre-check of App. A).
//   reduce_kernel  O(N): fixed-order sum of the partial accelerations, scatter to
//                  the caller's order, optional v += dt * a (the Kick of App. A).
//
// No code, header, table or helper is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace genga {

#define GENGA_STATUS_COINCIDENT 1
// Padding records sit far from every real body; records used as i-bodies and as j-bodies share
// one array, so a padding i meets a padding j at distance 0 -- its lanes are never stored.
#define GENGA_SENTINEL_POS 1.0e15   // its square fits a float (group boxes are kept in FP32)
#define GENGA_CHUNK 8              // j-records per filter chunk (one warp vote per chunk)
#define GENGA_GROUP 32             // j-records per culling group (one box per group)
#define GENGA_PAD 1024             // record arrays are padded to multiples of this

struct KickParams {
    // records (library scratch), internal order: massive bodies in [0, m_pad), semi-active test
    // particles from m_pad on; padding records have idx = -1, G m = 0, filter word = -1
    const double2* __restrict__ rxy;   // (x, y)
    const double2* __restrict__ rzm;   // (z, G m)
    const int* __restrict__ rfw;       // filter word (see filter_word)
    const int* __restrict__ ridx;      // caller's body index, -1 for padding
    const float4* __restrict__ cblo;   // box of each group of GENGA_GROUP records: (lo x, lo y, lo z, max filter word)
    const float4* __restrict__ cbhi;   //                                            (hi x, hi y, hi z, -)
    // the caller's arrays (read by the exact per-pair path only)
    const double* __restrict__ rcrit;  // [L+1][N]
    int N, n_massive, L;
    int react;                         // TP 2 at level >= 1: exact_kernel also adds the reaction of a semi-active
                                       // particle i on the massive body j (near_kernel's pair filter is symmetric)
    int j_rec0;                        // record of the first j-tile (0; m_pad in the second pass of TP 2)
    int i_rec0;                        // record of the first i-block (0; m_pad for the particles' rows beside kick_sym_kernel)
    int i_rec_end;                     // i-records from here on take no part in the pass (n_rec; m_pad in the second pass
                                       // of TP 2, whose last i-block may reach past the massive records: sec. 8.1
                                       // particles never feel each other)
    int force_only;                    // second pass of TP 2 at level 0 (massive i x semi-active j): candidates are
                                       // queued as (i, ~j): exact_kernel adds the force on i and leaves the encounter
                                       // bookkeeping to the first pass, which meets the same pair from the particle's side
    double f;                          // enc_factor
    // decomposition (genga_kick_plan)
    int n_j_tiles, n_ctas, max_segs;
    long long n_tiles;
    double* __restrict__ partial;      // [n_ctas][max_segs][3][i_block]
    // encounter output
    int* __restrict__ out_pairs;       // [capacity][2]
    long long capacity;
    int* __restrict__ out_npairs;      // [N + 1]; nullptr: no pre-check output wanted (closing kick of genga_step)
    int* __restrict__ status;
    // exact path (candidate list, fixed-point accumulators)
    int2* __restrict__ cand;           // [cand_capacity] (i-record, j-record)
    long long cand_capacity;
    int* __restrict__ ncand;           // candidates appended (may exceed the capacity: status bit)
    unsigned long long* __restrict__ fx;   // [3][GENGA_FX_LIMBS][fx_stride], all zero between calls (a record's limbs lie
                                           // fx_stride apart: reduce_kernel reads them coalesced)
    long long fx_stride;
    int* __restrict__ touched;         // [n_rec] != 0: the record's accumulators were added to
    const int* __restrict__ need_near; // level >= 1 kick on the candidate list of the level-0 kick (GENGA_KICK_REUSE_LIST):
                                       // != 0 if that list may miss a pair of this level (pack_kernel); nullptr otherwise
};

// the candidate list cannot serve this kick: near_kernel<true> searches and evaluates all pairs itself
__device__ __forceinline__ bool list_unusable(const KickParams& p)
{
    return (long long)*p.ncand > p.cand_capacity || (p.need_near && *p.need_near != 0);
}

// ---------------------------------------------------------------------------------------------
// Filter word of a body.  With R_b = max(rc0_b, f rcL_b), a pair (i, j) can only have W != 1
// (level 0), W != 0 (level >= 1: the factor 1 - K_0 of eq. 63 PAPER.md:627-632 vanishes for
// r >= rc0_ij) or be an encounter pair (r < f rcL_ij) if r < max(R_i, R_j).  Positive doubles
// order like their bit patterns, so the test is done on the HIGH WORDS on the integer pipe
// (DSETP runs at a quarter of the DFMA rate); the + 1 covers the truncated low word, the one-ulp
// difference between the fused r^2 of the pair loop and the unfused r^2 of the exact path, and
// the rounding of y = (r - 0.1 rc)/(0.9 rc) near 1: a pair that passes the filter has
// hi(r^2) >= hi(R^2) + 1, i.e. r^2 exceeds R^2 by at least one unit of the high word minus the
// truncated low word of R^2 -- a margin between 1 ulp of the high word (2^-20 relative) and, when
// R^2's low word is all ones, a single ulp of the double.  Either is enough: r^2 > R^2 strictly in
// both the fused and the unfused evaluation means K = 1 (level 0) resp. 1 - K_0 = 0 and no encounter.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ int filter_word(double rc0, double rcL, double f, double scale)
{
    // scale = 1 but for the merged kick of consecutive steps (genga_kick_merged), whose candidate list must also
    // hold the pairs inside the critical radii of the NEXT step, not known yet: they may be larger by that factor
    const double m = __dmul_rn(fmax(rc0, __dmul_rn(f, rcL)), scale);
    return __double2hiint(__dmul_rn(m, m)) + 1;
}

// perm == nullptr: internal order = caller's order; else perm[s] = caller's index of the body at
// sorted position s (massive bodies first).  One warp writes one group of GENGA_GROUP records and
// its bounding box (FP32, rounded outwards).
__global__ void __launch_bounds__(256)
pack_kernel(const double* __restrict__ pos, const double* __restrict__ mass, const double* __restrict__ rcrit,
            const int* __restrict__ perm, int N, int n_massive, int m_pad, int n_rec, int L, double G, double f,
            double fw_scale, double2* __restrict__ rxy, double2* __restrict__ rzm, int* __restrict__ rfw, int* __restrict__ ridx,
            float4* __restrict__ cblo, float4* __restrict__ cbhi, int* __restrict__ out_npairs,
            int* __restrict__ ncand, int* __restrict__ rfw_ref, int* __restrict__ need_near, int n_levels, int keep_list)
{
    // keep_list (GENGA_KICK_REUSE_LIST, level >= 1): the candidate list of the level-0 kick stays; a body whose filter
    // word now exceeds the one that list was built with (rfw_ref) raises need_near[L].  The level-0 kick writes rfw_ref
    // and clears the flags of every level.
    if (blockIdx.x == 0 && threadIdx.x == 0 && !keep_list) *ncand = 0;
    if (blockIdx.x == 0 && rfw_ref && !keep_list)
        for (int l = threadIdx.x; l < n_levels; l += blockDim.x) need_near[l] = 0;
    const int stride = gridDim.x * blockDim.x;       // a multiple of 32
    const int top = max(n_rec, ((N + 1 + 31) / 32) * 32);
    for (int r = blockIdx.x * blockDim.x + threadIdx.x; r < top; r += stride) {
        int fw = -1;
        double x = GENGA_SENTINEL_POS, y = GENGA_SENTINEL_POS, z = GENGA_SENTINEL_POS, gm = 0.0;
        if (r < n_rec) {
            int b = -1;                               // caller's index of record r
            if (r < m_pad) { if (r < n_massive) b = r; }
            else if (r - m_pad < N - n_massive) b = n_massive + (r - m_pad);
            if (b >= 0 && perm) b = perm[b];
            if (b >= 0) {
                x = pos[b]; y = pos[(size_t)N + b]; z = pos[2 * (size_t)N + b];
                gm = __dmul_rn(G, mass[b]);
                fw = filter_word(rcrit[b], rcrit[(size_t)L * N + b], f, fw_scale);
            }
            rxy[r] = make_double2(x, y);
            rzm[r] = make_double2(z, gm);
            rfw[r] = fw;
            ridx[r] = b;
            if (rfw_ref) {
                if (!keep_list) rfw_ref[r] = fw;
                else if (fw > rfw_ref[r]) need_near[L] = 1;
            }
        }
        int m = fw;
        // group box
        // ... over the real bodies of the group only: a padding record (fw = -1) cannot trip the
        // filter, and a group without real bodies gets an empty box that is near to nothing
        const bool real = fw >= 0;
        float lx = real ? __double2float_rd(x) : 3.0e38f, ly = real ? __double2float_rd(y) : 3.0e38f,
              lz = real ? __double2float_rd(z) : 3.0e38f;
        float hx = real ? __double2float_ru(x) : -3.0e38f, hy = real ? __double2float_ru(y) : -3.0e38f,
              hz = real ? __double2float_ru(z) : -3.0e38f;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, o));
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            lx = fminf(lx, __shfl_xor_sync(0xffffffffu, lx, o)); hx = fmaxf(hx, __shfl_xor_sync(0xffffffffu, hx, o));
            ly = fminf(ly, __shfl_xor_sync(0xffffffffu, ly, o)); hy = fmaxf(hy, __shfl_xor_sync(0xffffffffu, hy, o));
            lz = fminf(lz, __shfl_xor_sync(0xffffffffu, lz, o)); hz = fmaxf(hz, __shfl_xor_sync(0xffffffffu, hz, o));
        }
        if (r < n_rec && (r % GENGA_GROUP) == 0) {
            cblo[r / GENGA_GROUP] = make_float4(lx, ly, lz, __int_as_float(m));
            cbhi[r / GENGA_GROUP] = make_float4(hx, hy, hz, 0.0f);
        }
        if (out_npairs && r <= N) out_npairs[r] = 0;
    }
}

// ---------------------------------------------------------------------------------------------
// The changeover function K (form of Chambers 1999 eq. 10, reading G1 of
// DESIGN.md), evaluated with IEEE operations in a fixed order and no contraction.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ double changeover_K(double r, double rc)
{
    const double y = __ddiv_rn(__dsub_rn(r, __dmul_rn(0.1, rc)), __dmul_rn(0.9, rc));
    if (y <= 0.0) return 0.0;
    if (y >= 1.0) return 1.0;
    const double yy = __dmul_rn(y, y);
    const double twoy = __dmul_rn(2.0, y);
    const double den = __dadd_rn(__dsub_rn(__dmul_rn(twoy, y), twoy), 1.0);
    return __ddiv_rn(yy, den);
}

struct ExactResult {
    double s;     // G m_j W_L / r^3 (0 if the pair contributes nothing)
    double W;     // W_L
    double r3;    // r^2 * r
    int enc;      // 1 if (i, j) is an encounter pair
};

// The exact per-pair evaluation for the few pairs the filter lets through: the level weight W_L
// and the pre-check, in unfused IEEE arithmetic (so the strict comparison r^2 < (f rcL)^2 is taken
// on the bits a plain left-to-right evaluation gives).  Out of line: it runs for ~1e-4 of the
// pairs and must not cost the pair loop registers.  bi, bj are the caller's indices.
__device__ __noinline__ ExactResult exact_pair(const double* __restrict__ rcrit, int N, int L, double f, int* status,
                                               int bi, int bj, double dx, double dy, double dz, double gmj)
{
    ExactResult out;
    out.s = 0.0;
    out.W = 0.0;
    out.r3 = 1.0;
    out.enc = 0;
    const double r2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
    if (!(r2 > 0.0)) {                                             // coincident distinct bodies
        atomicOr(status, GENGA_STATUS_COINCIDENT);
        return out;
    }
    const double r = __dsqrt_rn(r2);
    const size_t n = (size_t)N;
    const double rcL = fmax(rcrit[L * n + bi], rcrit[L * n + bj]);
    const double thr = __dmul_rn(f, rcL);
    out.enc = r2 < __dmul_rn(thr, thr) ? 1 : 0;
    double W = 1.0;
    for (int k = 0; k < L; k++) {
        const double rck = fmax(rcrit[k * n + bi], rcrit[k * n + bj]);
        W = __dmul_rn(W, __dsub_rn(1.0, changeover_K(r, rck)));
    }
    W = __dmul_rn(W, changeover_K(r, rcL));
    out.W = W;
    out.r3 = __dmul_rn(r2, r);
    if (W != 0.0) out.s = __ddiv_rn(__dmul_rn(gmj, W), out.r3);
    return out;
}

// ---------------------------------------------------------------------------------------------
// mbarrier + 1-D TMA bulk copy (cp.async.bulk, SASS UBLKCP) for the j-tile staging
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t phase)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@!p bra WAIT_%=;\n\t}"
        ::"r"(smem_u32(bar)), "r"(phase) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

// MUFU.RSQ64H: 1/sqrt to ~2^-20 from the high word only (low word of the result is 0); runs on
// the SFU pipe, not the FP64 pipe.  Skipped (result 0) for pairs the filter catches, so that they
// add exactly 0 in the pair loop and r2 = 0 (the self pair) never makes an infinity.
__device__ __forceinline__ double rsqrt_seed_unless(double x, bool skip)
{
    double y = 0.0;
    asm("{\n\t.reg .pred q;\n\tsetp.ne.s32 q, %2, 0;\n\t@!q rsqrt.approx.ftz.f64 %0, %1;\n\t}"
        : "+d"(y) : "d"(x), "r"((int)skip));
    return y;
}

// ---------------------------------------------------------------------------------------------
// The pair loop's arithmetic for one (i, j) -- ROW a2-a4 of SURVEY.md section 8(a).
//   d = x_j - x_i, r2 = d.d                         3 DADD, 1 DMUL, 2 DFMA
//   trig = hi(r2) < thr  (integer pipe)             the pair goes to the exact path instead
//   level 0 (W = K = 1 for every pair that passes the filter):
//     y0 = MUFU.RSQ64H(r2) ~ r^-1 (1 + O(2^-20));  e = 1 - r2 y0^2
//     G m_j r^-3 = y0^2 (G m_j y0) (1 + e (3/2 + 15/8 e))  + O(e^3)      4 DMUL, 3 DFMA
//     a += s d                                       3 DFMA
//   16 FP64-pipe instructions, 24 flops.  Every DFMA but the three accumulations has at most two
//   distinct register operands (a third costs a register-file cycle on this part).
//   (level >= 1: a pair that passes the filter has W_L = 0 exactly -- near_kernel, no arithmetic.)
// ---------------------------------------------------------------------------------------------
// The same arithmetic without the filter, for groups the box test has cleared.
__device__ __forceinline__ void pair_bare(double xj, double yj, double zj, double gmj,
                                          double xi, double yi, double zi, double& ax, double& ay, double& az)
{
    const double dx = __dsub_rn(xj, xi), dy = __dsub_rn(yj, yi), dz = __dsub_rn(zj, zi);
    const double r2 = fma(dz, dz, fma(dy, dy, __dmul_rn(dx, dx)));
    double y0;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y0) : "d"(r2));
    const double t = __dmul_rn(y0, y0);
    const double e = fma(-r2, t, 1.0);
    const double g = __dmul_rn(gmj, y0);
    const double u = __dmul_rn(t, g);
    const double c = fma(1.875, e, 1.5);
    const double q = fma(e, c, 1.0);
    const double s = __dmul_rn(u, q);
    ax = fma(s, dx, ax);
    ay = fma(s, dy, ay);
    az = fma(s, dz, az);
}

__device__ __forceinline__ void pair_fast(double xj, double yj, double zj, double gmj,
                                          double xi, double yi, double zi, int thr,
                                          double& ax, double& ay, double& az, bool& any)
{
    const double dx = __dsub_rn(xj, xi), dy = __dsub_rn(yj, yi), dz = __dsub_rn(zj, zi);
    const double r2 = fma(dz, dz, fma(dy, dy, __dmul_rn(dx, dx)));
    const bool trig = __double2hiint(r2) < thr;
    any |= trig;
    const double y0 = rsqrt_seed_unless(r2, trig);
    const double t = __dmul_rn(y0, y0);
    const double e = fma(-r2, t, 1.0);
    const double g = __dmul_rn(gmj, y0);
    const double u = __dmul_rn(t, g);
    const double c = fma(1.875, e, 1.5);
    const double q = fma(e, c, 1.0);
    const double s = __dmul_rn(u, q);
    ax = fma(s, dx, ax);
    ay = fma(s, dy, ay);
    az = fma(s, dz, az);
}

// ---------------------------------------------------------------------------------------------
// kick_kernel.  CTA c owns the tiles [c T / C, (c+1) T / C) of the i-major (i-block x j-tile)
// grid (genga_kick_plan); warp w owns the 32 * IPT consecutive i-records
// ib * IB + w * 32 * IPT + [0, 32 * IPT), lane l the records k * 32 + l of them.
// j-tiles are staged by TMA bulk copies into a two-stage shared-memory ring; every lane reads
// the same j-record (LDS broadcast).
//
// Culling: per tile, lane g tests the box of the warp's i-records against the box of j-group g
// (GENGA_GROUP records).  If the boxes are further apart than the largest filter radius of either
// side, no pair of the (warp, group) combination can trip the filter, and the group runs the bare
// pair loop (no compare, no vote) -- same arithmetic, same order, same bits as the checked loop
// would give.  Otherwise the group runs the checked loop: per chunk of GENGA_CHUNK j-records one warp vote
// decides whether any pair of the chunk needs the exact path.
// ---------------------------------------------------------------------------------------------
template <int JT>
struct alignas(128) TileStage {
    double2 xy[JT];
    double2 zm[JT];
    float4 blo[JT / GENGA_GROUP];
    float4 bhi[JT / GENGA_GROUP];
    int fw[JT];
};

// lower bound of the squared distance between two boxes against the upper bound of the squared
// filter radius: true if some pair might trip the filter
__device__ __forceinline__ bool boxes_near(float4 alo, float4 ahi, int afw, float4 blo, float4 bhi)
{
    const float gx = fmaxf(fmaxf(__fsub_rd(alo.x, bhi.x), __fsub_rd(blo.x, ahi.x)), 0.0f);
    const float gy = fmaxf(fmaxf(__fsub_rd(alo.y, bhi.y), __fsub_rd(blo.y, ahi.y)), 0.0f);
    const float gz = fmaxf(fmaxf(__fsub_rd(alo.z, bhi.z), __fsub_rd(blo.z, ahi.z)), 0.0f);
    const float d2 = __fmaf_rd(gx, gx, __fmaf_rd(gy, gy, __fmul_rd(gz, gz)));
    const int fw = max(max(afw, __float_as_int(blo.w)), 0);
    // the filter trips iff hi(r2) < fw, so r2 >= double(fw, 0) is safe; 1.0001 covers the FP32
    // roundings here and the ulp between the true and the computed r2
    const float R2 = __fmul_ru(__double2float_ru(__hiloint2double(fw, 0)), 1.0001f);
    return !(d2 >= R2);
}

// ---------------------------------------------------------------------------------------------
// Exact path, decoupled from the pair loop.  kick_kernel only APPENDS the pairs the filter catches
// to a global candidate list (ordered pairs (i-record, j-record); one atomic per warp and push);
// exact_kernel then evaluates one candidate per thread -- weight, pre-check, pair emission, counts.
// The candidates cluster where the disk is dense (inner edge: > 100 partners per body against a
// mean of 15), so evaluating them where they are found serialises a few warps; as a list they
// spread over the whole device.
//
// The candidates' terms G m_j W d / r^3 are added to body i in FIXED POINT: integer addition is
// associative, so the sum does not depend on the (arbitrary) order of the list and every output
// bit stays a fixed function of the inputs.  A body's accumulator is, per
// component, GENGA_FX_LIMBS 64-bit integers; limb l counts units of 2^(GENGA_FX_E0 + 32 l).  A
// double is cut into three 32-bit pieces on that grid (exactly, unless bits fall below
// 2^GENGA_FX_E0: those are truncated towards zero) and each piece is added with one 64-bit
// integer atomic; a limb has room for 2^31 pieces.  reduce_kernel propagates the carries,
// rounds the 96 leading bits to a double and adds it to the far-field sum.
// Window: [2^-140, 2^52) = [7e-43, 4.5e15] AU/day^2.
// ---------------------------------------------------------------------------------------------
#define GENGA_FX_LIMBS 6
#define GENGA_FX_E0 (-140)
#define GENGA_STATUS_CAND_OVERFLOW 2
#define GENGA_STATUS_FX_RANGE 4

__device__ __forceinline__ void fx_add(unsigned long long* __restrict__ acc, long long stride, double x, int* status)
{
    const long long bits = __double_as_longlong(x);
    const int ex = (int)((bits >> 52) & 0x7ff);
    unsigned long long m = (unsigned long long)bits & 0xfffffffffffffULL;
    if (ex == 0x7ff) { atomicOr(status, GENGA_STATUS_FX_RANGE); return; }      // inf / nan
    int e = -1074;                                                              // x = +- m 2^e
    if (ex) { m |= 1ULL << 52; e = ex - 1075; }
    int pos = e - GENGA_FX_E0;                                                  // grid position of m's lowest bit
    if (pos < 0) {
        if (pos <= -53) return;
        m >>= -pos;
        pos = 0;
    }
    if (m == 0) return;
    const int l0 = pos >> 5, r = pos & 31;
    const unsigned long long lo = m << r;
    const unsigned long long q0 = lo & 0xffffffffULL, q1 = lo >> 32, q2 = r ? (m >> (64 - r)) : 0ULL;
    const bool neg = bits < 0;
    if ((q0 && l0 >= GENGA_FX_LIMBS) || (q1 && l0 + 1 >= GENGA_FX_LIMBS) || (q2 && l0 + 2 >= GENGA_FX_LIMBS)) {
        atomicOr(status, GENGA_STATUS_FX_RANGE);
        return;
    }
    if (q0) atomicAdd(acc + l0 * stride, neg ? 0ULL - q0 : q0);
    if (q1) atomicAdd(acc + (l0 + 1) * stride, neg ? 0ULL - q1 : q1);
    if (q2) atomicAdd(acc + (l0 + 2) * stride, neg ? 0ULL - q2 : q2);
}

// value of one accumulator; clears it for the next call
__device__ __forceinline__ double fx_take(unsigned long long* __restrict__ acc, long long stride, int* status)
{
    unsigned w[GENGA_FX_LIMBS];
    long long carry = 0;
#pragma unroll
    for (int l = 0; l < GENGA_FX_LIMBS; l++) {
        const long long v = (long long)acc[l * stride] + carry;
        acc[l * stride] = 0ULL;
        w[l] = (unsigned)((unsigned long long)v & 0xffffffffULL);
        carry = v >> 32;                                   // arithmetic: the sign travels upwards
    }
    if (carry != 0 && carry != -1) atomicOr(status, GENGA_STATUS_FX_RANGE);
    const bool neg = carry < 0;
    if (neg) {                                             // two's complement -> magnitude
        unsigned c = 1u;
#pragma unroll
        for (int l = 0; l < GENGA_FX_LIMBS; l++) {
            const unsigned t = ~w[l];
            w[l] = t + c;
            c = (c && t == 0xffffffffu) ? 1u : 0u;
        }
    }
    int h = -1;
#pragma unroll
    for (int l = 0; l < GENGA_FX_LIMBS; l++)
        if (w[l]) h = l;
    if (h < 0) return 0.0;
    double v = 0.0;                                        // the three leading limbs
#pragma unroll
    for (int l = GENGA_FX_LIMBS - 1; l >= 0; l--)
        if (l <= h && l >= h - 2) v = __dadd_rn(__dmul_rn(v, 4294967296.0), (double)w[l]);
    const int lowest = h >= 2 ? h - 2 : 0;
    v = scalbn(v, GENGA_FX_E0 + 32 * lowest);
    return neg ? -v : v;
}

// The work of the exact path for one candidate (i-record, j-record or ~j-record for a force-only
// candidate, or (-1, -1) for an empty slot): weight, force on i (and the TP 2 reaction on j), pre-check,
// per-body counts.  Returns the pair to emit, if any.
__device__ __forceinline__ void apply_candidate(const KickParams& p, int ir_enc, int jr_enc, bool& hit, int& lo, int& hi)
{
    // (i, j) one-sided: the force on i and i's side of the bookkeeping (the mirror (j, i) is queued too);
    // (i, ~j) force-only: see KickParams;  (~i, j) symmetric (kick_sym_kernel): both forces, the pair's bookkeeping once;
    // (-1, -1) an empty slot
    const bool sym = ir_enc < 0 && jr_enc >= 0;
    const int ir = sym ? ~ir_enc : ir_enc;
    const bool force_only = ir >= 0 && jr_enc < 0;
    const int jr = force_only ? ~jr_enc : jr_enc;
    const int bi = ir >= 0 ? p.ridx[ir] : -1, bj = ir >= 0 ? p.ridx[jr] : -1;      // (-1, -1): empty slot
    if (ir == jr || bi < 0 || bj < 0) return;
    if (force_only && bi >= p.n_massive) return;            // the second pass of TP 2 only serves massive i
    if (force_only && p.L > 0) return;                      // a level-0 list at level >= 1: `react` covers TP 2 there
    const double2 ixy = p.rxy[ir], izm = p.rzm[ir], jxy = p.rxy[jr], jzm = p.rzm[jr];
    const double dx = __dsub_rn(jxy.x, ixy.x), dy = __dsub_rn(jxy.y, ixy.y), dz = __dsub_rn(jzm.x, izm.x);
    const ExactResult r = exact_pair(p.rcrit, p.N, p.L, p.f, p.status, bi, bj, dx, dy, dz, jzm.y);
    if (r.s != 0.0) {
        unsigned long long* acc = p.fx + ir;
        fx_add(acc, p.fx_stride, __dmul_rn(r.s, dx), p.status);
        fx_add(acc + GENGA_FX_LIMBS * p.fx_stride, p.fx_stride, __dmul_rn(r.s, dy), p.status);
        fx_add(acc + 2 * GENGA_FX_LIMBS * p.fx_stride, p.fx_stride, __dmul_rn(r.s, dz), p.status);
        p.touched[ir] = 1;
    }
    if (sym && r.W != 0.0 && izm.y != 0.0) {
        // the force of i on j with the bits the definition gives from j's side (d -> -d, r^2 and W unchanged)
        const double si = __ddiv_rn(__dmul_rn(izm.y, r.W), r.r3);
        unsigned long long* accj = p.fx + jr;
        fx_add(accj, p.fx_stride, -__dmul_rn(si, dx), p.status);
        fx_add(accj + GENGA_FX_LIMBS * p.fx_stride, p.fx_stride, -__dmul_rn(si, dy), p.status);
        fx_add(accj + 2 * GENGA_FX_LIMBS * p.fx_stride, p.fx_stride, -__dmul_rn(si, dz), p.status);
        p.touched[jr] = 1;
    }
    if (p.react && bi >= p.n_massive && r.W != 0.0 && izm.y != 0.0) {
        // TP 2: the reaction of the semi-active particle i on the massive body j, G m_i W (x_i - x_j) / r^3,
        // with the bits the definition gives from j's side (d -> -d, r^2 unchanged)
        const double si = __ddiv_rn(__dmul_rn(izm.y, r.W), r.r3);
        unsigned long long* accj = p.fx + jr;
        fx_add(accj, p.fx_stride, -__dmul_rn(si, dx), p.status);
        fx_add(accj + GENGA_FX_LIMBS * p.fx_stride, p.fx_stride, -__dmul_rn(si, dy), p.status);
        fx_add(accj + 2 * GENGA_FX_LIMBS * p.fx_stride, p.fx_stride, -__dmul_rn(si, dz), p.status);
        p.touched[jr] = 1;
    }
    if (r.enc && p.out_npairs && !force_only) {
        atomicAdd(p.out_npairs + bi, 1);
        if (sym) {                             // both massive, queued once
            atomicAdd(p.out_npairs + bj, 1);
            hit = true; lo = min(bi, bj); hi = max(bi, bj);
        } else if (bi >= p.n_massive) {        // test particle i, massive j
            atomicAdd(p.out_npairs + bj, 1);
            hit = true; lo = bj; hi = bi;
        } else if (bi < bj) {
            hit = true; lo = bi; hi = bj;
        }
    }
}

// Append the warp's tripped pairs (i-record, j-record) to the candidate list.  A warp reserves the
// list GENGA_CAND_BLOCK slots at a time (one atomic per block, not per push: the counter is a
// single hot address) and fills its block with a private cursor; the slots of a block it does
// not use are closed with the empty entry (-1, -1), which exact_kernel skips.
#define GENGA_CAND_BLOCK 128

struct CandCursor {
    long long base;   // first slot of the warp's open block (warp-uniform)
    int fill;         // slots used in it; GENGA_CAND_BLOCK: no block open
    bool over;        // the warp has seen the list full: it reserves no more (the counter stays below
                      // capacity + one block per warp of the grid and cannot wrap); see near_kernel<true>
};

__device__ __forceinline__ void close_block(const KickParams& p, CandCursor& c)
{
    const int lane = threadIdx.x & 31;
    for (int q = c.fill + lane; q < GENGA_CAND_BLOCK; q += 32)
        if (c.base + q < p.cand_capacity) p.cand[c.base + q] = make_int2(-1, -1);
    c.fill = GENGA_CAND_BLOCK;
}

__device__ __forceinline__ void push_candidates(const KickParams& p, CandCursor& c, bool mine, int irec, int jrec)
{
    const unsigned m = __ballot_sync(0xffffffffu, mine);
    if (c.over) return;                                     // warp-uniform; the list is abandoned (near_kernel<true>)
    const int lane = threadIdx.x & 31;
    const int n = __popc(m);
    if (c.fill + n > GENGA_CAND_BLOCK) {                    // warp-uniform
        if (c.fill < GENGA_CAND_BLOCK) close_block(p, c);
        int base = 0;
        if (lane == 0) {
            base = atomicAdd(p.ncand, GENGA_CAND_BLOCK);
            if ((long long)base + GENGA_CAND_BLOCK > p.cand_capacity) atomicOr(p.status, GENGA_STATUS_CAND_OVERFLOW);
        }
        c.base = __shfl_sync(0xffffffffu, base, 0);
        c.fill = 0;
        if (c.base < 0 || c.base + GENGA_CAND_BLOCK > p.cand_capacity) {      // *ncand > capacity from now on
            c.over = true;
            c.fill = GENGA_CAND_BLOCK;
            return;
        }
    }
    if (mine) {
        const long long slot = c.base + c.fill + __popc(m & ((1u << lane) - 1u));
        if (slot >= 0 && slot < p.cand_capacity) p.cand[slot] = make_int2(irec, jrec);
    }
    c.fill += n;
}

// Emission for a whole CTA of 256 threads with U candidates per thread: ONE atomic on the pair counter
// per CTA and round (the counter is a single address, and an atomic that returns a value waits for it:
// one per warp made exact_kernel wait ~30,000 times in a row on that address at N = 65,536).
#define GENGA_EXACT_U 4

template <int U>
__device__ __forceinline__ void emit_pairs_cta(const KickParams& p, const bool (&hit)[U], const int (&lo)[U],
                                               const int (&hi)[U])
{
    __shared__ int wsum[8];
    __shared__ int cta_base;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int mine = 0;
#pragma unroll
    for (int u = 0; u < U; u++) mine += hit[u] ? 1 : 0;
    int s = mine;                                           // inclusive scan over the warp
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, s, o);
        if (lane >= o) s += t;
    }
    if (lane == 31) wsum[warp] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        int tot = 0;
#pragma unroll
        for (int w = 0; w < 8; w++) { const int c = wsum[w]; wsum[w] = tot; tot += c; }
        cta_base = tot ? atomicAdd(p.out_npairs + p.N, tot) : 0;
    }
    __syncthreads();
    long long slot = (long long)cta_base + wsum[warp] + (s - mine);
#pragma unroll
    for (int u = 0; u < U; u++)
        if (hit[u]) {
            if (slot < p.capacity) reinterpret_cast<int2*>(p.out_pairs)[slot] = make_int2(lo[u], hi[u]);
            slot++;
        }
    __syncthreads();                                        // wsum / cta_base are reused by the next round
}

__global__ void __launch_bounds__(256) exact_kernel(const KickParams p)
{
    constexpr int U = GENGA_EXACT_U;
    if (list_unusable(p)) return;                           // the list overflowed: near_kernel<true> has done all of it
    const long long n = (long long)*p.ncand;
    // a CTA walks the list in rounds of 256 * U candidates (CTA-uniform trip count: the emission synchronises)
    for (long long cbase = (long long)blockIdx.x * (256 * U); cbase < n; cbase += (long long)gridDim.x * (256 * U)) {
        bool hit[U];
        int lo[U], hi[U];
#pragma unroll
        for (int u = 0; u < U; u++) {
            const long long c = cbase + u * 256 + threadIdx.x;
            hit[u] = false; lo[u] = 0; hi[u] = 0;
            if (c >= n) continue;
            const int2 e = p.cand[c];
            apply_candidate(p, e.x, e.y, hit[u], lo[u], hi[u]);
        }
        emit_pairs_cta<U>(p, hit, lo, hi);
    }
}

__device__ __forceinline__ void mbar_arrive(uint64_t* bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}


template <int THREADS, int IPT, int JT, int CTAS, int STAGES>
__global__ void __launch_bounds__(THREADS, CTAS) kick_kernel(const KickParams p)
{
    constexpr int IB = THREADS * IPT;
    constexpr int WARPS = THREADS / 32;
    constexpr int NG = JT / GENGA_GROUP;
    constexpr uint32_t TILE_BYTES = JT * 32 + NG * 32 + JT * 4;
    static_assert(NG <= 32 && JT % GENGA_GROUP == 0, "one lane per group");
    static_assert(GENGA_CHUNK * IPT <= 32, "one trigger bit per pair of a chunk");
    __shared__ TileStage<JT> st[STAGES];
    __shared__ __align__(8) uint64_t full[STAGES];
    __shared__ __align__(8) uint64_t empty[STAGES];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int woff = warp * (32 * IPT) + lane;              // offset of the thread's first record in the i-block
    const long long t0 = plan_tile_begin(blockIdx.x, p.n_tiles, p.n_ctas);
    const long long t1 = plan_tile_begin(blockIdx.x + 1, p.n_tiles, p.n_ctas);
    if (t0 >= t1) return;

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < STAGES; s++) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], WARPS);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    // tile t0 + g goes to stage g % STAGES; the stage is free once every warp has arrived on its
    // `empty` barrier for the tile that used it before (g - STAGES)
    auto issue = [&](int g) {
        const int s = g % STAGES;
        if (g >= STAGES) mbar_wait(&empty[s], (uint32_t)((g / STAGES - 1) & 1));
        const int jt = (int)((t0 + g) % p.n_j_tiles);
        mbar_expect_tx(&full[s], TILE_BYTES);
        const size_t j0 = (size_t)p.j_rec0 + (size_t)jt * JT;          // a multiple of 64: every offset 16-byte aligned
        bulk_g2s(st[s].xy, p.rxy + j0, JT * 16, &full[s]);
        bulk_g2s(st[s].zm, p.rzm + j0, JT * 16, &full[s]);
        bulk_g2s(st[s].blo, p.cblo + j0 / GENGA_GROUP, NG * 16, &full[s]);
        bulk_g2s(st[s].bhi, p.cbhi + j0 / GENGA_GROUP, NG * 16, &full[s]);
        bulk_g2s(st[s].fw, p.rfw + j0, JT * 4, &full[s]);
    };
    const int n_it = (int)(t1 - t0);
    if (tid == 0)
        for (int g = 0; g < STAGES && g < n_it; g++) issue(g);

    double xi[IPT], yi[IPT], zi[IPT], ax[IPT], ay[IPT], az[IPT];
    int fi[IPT];
    float4 wlo, whi;                                        // box of the warp's i-records
    int wfw = -1;
    const int first_ib = (int)(t0 / p.n_j_tiles);
    int cur_ib = -1;
    CandCursor cc;
    cc.base = 0;
    cc.fill = GENGA_CAND_BLOCK;
    cc.over = false;

    auto flush = [&]() {
        const size_t base = ((size_t)blockIdx.x * p.max_segs + (cur_ib - first_ib)) * 3 * IB;
#pragma unroll
        for (int k = 0; k < IPT; k++) {
            const int off = woff + k * 32;
            p.partial[base + off] = ax[k];
            p.partial[base + IB + off] = ay[k];
            p.partial[base + 2 * IB + off] = az[k];
        }
    };

    for (int it = 0; it < n_it; ++it) {
        const long long t = t0 + it;
        const int s = it % STAGES;
        const int ib = (int)(t / p.n_j_tiles);
        const int jt = (int)(t - (long long)ib * p.n_j_tiles);
        if (ib != cur_ib) {
            if (cur_ib >= 0) flush();
            cur_ib = ib;
            wlo = make_float4(3.0e38f, 3.0e38f, 3.0e38f, 0.0f);
            whi = make_float4(-3.0e38f, -3.0e38f, -3.0e38f, 0.0f);
            wfw = -1;
#pragma unroll
            for (int k = 0; k < IPT; k++) {
                const size_t r = (size_t)p.i_rec0 + (size_t)ib * IB + woff + k * 32;
                ax[k] = ay[k] = az[k] = 0.0;
                if (r >= (size_t)p.i_rec_end) {             // whole groups of 32 records (i_rec_end is a multiple of 32)
                    xi[k] = yi[k] = zi[k] = GENGA_SENTINEL_POS;
                    fi[k] = -1;
                    continue;
                }
                const double2 a = p.rxy[r], b = p.rzm[r];
                xi[k] = a.x; yi[k] = a.y; zi[k] = b.x;
                fi[k] = p.rfw[r];
                // the groups of GENGA_GROUP records are aligned with the warp's k-slices
                const float4 glo = p.cblo[r / GENGA_GROUP], ghi = p.cbhi[r / GENGA_GROUP];
                wlo.x = fminf(wlo.x, glo.x); wlo.y = fminf(wlo.y, glo.y); wlo.z = fminf(wlo.z, glo.z);
                whi.x = fmaxf(whi.x, ghi.x); whi.y = fmaxf(whi.y, ghi.y); whi.z = fmaxf(whi.z, ghi.z);
                wfw = max(wfw, __float_as_int(glo.w));
            }
        }
        mbar_wait(&full[s], (uint32_t)((it / STAGES) & 1));
        const TileStage<JT>& S = st[s];

        const bool mine_near = lane < NG ? boxes_near(wlo, whi, wfw, S.blo[lane], S.bhi[lane]) : false;
        const unsigned nearmask = __ballot_sync(0xffffffffu, mine_near);

#pragma unroll 1
        for (int g = 0; g < NG; g++) {
            const int j0 = g * GENGA_GROUP;
            if (!((nearmask >> g) & 1u)) {
#pragma unroll 4
                for (int u = 0; u < GENGA_GROUP; u++) {
                    const double2 xy = S.xy[j0 + u], zm = S.zm[j0 + u];
#pragma unroll
                    for (int k = 0; k < IPT; k++)
                        pair_bare(xy.x, xy.y, zm.x, zm.y, xi[k], yi[k], zi[k], ax[k], ay[k], az[k]);
                }
                continue;
            }
#pragma unroll 1
            for (int jj = j0; jj < j0 + GENGA_GROUP; jj += GENGA_CHUNK) {
                unsigned tm = 0;                            // bit u * IPT + k: pair (k, jj + u) tripped the filter
#pragma unroll
                for (int u = 0; u < GENGA_CHUNK; u++) {
                    const double2 xy = S.xy[jj + u], zm = S.zm[jj + u];
                    const int fj = S.fw[jj + u];            // the exact per-pair rule: hi(r^2) < max(fw_i, fw_j)
#pragma unroll
                    for (int k = 0; k < IPT; k++) {
                        bool trig = false;
                        pair_fast(xy.x, xy.y, zm.x, zm.y, xi[k], yi[k], zi[k], max(fi[k], fj), ax[k], ay[k], az[k], trig);
                        tm |= (trig ? 1u : 0u) << (u * IPT + k);
                    }
                }
                unsigned todo = __reduce_or_sync(0xffffffffu, tm);
                while (todo) {                              // warp-uniform: the (u, k) some lane tripped
                    const int b = __ffs(todo) - 1;
                    todo &= todo - 1;
                    const bool mine = (tm >> b) & 1u;
                    const int jrec = p.j_rec0 + jt * JT + jj + b / IPT;
                    push_candidates(p, cc, mine, p.i_rec0 + ib * IB + woff + (b % IPT) * 32, p.force_only ? ~jrec : jrec);
                }
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[s]);              // this warp is done with stage s
        if (tid == 0 && it >= 1 && it - 1 + STAGES < n_it) issue(it - 1 + STAGES);
    }
    flush();
    if (cc.fill < GENGA_CAND_BLOCK) close_block(p, cc);
}

// ---------------------------------------------------------------------------------------------
// near_kernel: the pair loop of changeover levels L >= 1.  The factor 1 - K_0 of eq. 63
// vanishes for r >= rc0_ij, so every pair that passes the filter has W_L = 0
// EXACTLY and is no encounter pair: the level-L kick is a neighbour search.  A warp owns one group
// of GENGA_GROUP i-records (one per lane) and tests its box against the box of every j-group
// (staged through shared memory GENGA_NEAR_BOXES at a time, one box per lane and vote); only for
// the few near groups it forms r^2 for its 32 x 32 pairs and appends the pairs that trip the
// filter to the candidate list.  No accelerations are accumulated here: all of them come from
// exact_kernel's fixed-point sums (reduce_kernel is told there are no partial segments).
// The near groups of a warp cluster where the disk is dense (a few warps have ten times the mean), and
// a warp walks its near groups one after the other: the j-groups are therefore dealt round-robin to
// gridDim.y CTAs per i-chunk (CTA y takes the groups g = y mod gridDim.y), which cuts the longest
// chain by that factor.
// ---------------------------------------------------------------------------------------------
#define GENGA_NEAR_THREADS 128
#define GENGA_NEAR_BOXES 256

// RESCAN = false: the level >= 1 pair loop (queues candidates; a pair trips if hi(r^2) < max(fw_i, fw_j)).
// RESCAN = true : the fallback for a candidate list that overflowed (more pairs inside critical radii than
//   the list holds: everything inside everything's radius).  Launched after the pair loop of every kick, it
//   returns at once unless the list overflowed; then it repeats the search -- with the pair loops' own trip
//   rule on the same bits (r^2 of (i, j) and of (j, i) are the same double), so that it meets exactly the ordered
//   pairs the far-field pass left out -- and evaluates every tripped pair where it finds it (apply_candidate), while
//   exact_kernel ignores the truncated list.  Slow (one atomic on the pair counter per pair) but complete:
//   the capacity of the list bounds the speed of pathological inputs, not the correctness of the result.
//   i-records [0, i_rec_end) against the j-groups [j_group0, j_group0 + n_jgroups); force_only as in KickParams.
template <bool RESCAN>
__global__ void __launch_bounds__(GENGA_NEAR_THREADS, 4)
near_kernel(const KickParams p, int i_rec_end, int j_group0, int n_jgroups, int force_only)
{
    if (RESCAN && !list_unusable(p)) return;
    __shared__ float4 blo[GENGA_NEAR_BOXES];
    __shared__ float4 bhi[GENGA_NEAR_BOXES];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int ig = blockIdx.x * (GENGA_NEAR_THREADS / 32) + warp;
    const int r = ig * GENGA_GROUP + lane;
    double xi = GENGA_SENTINEL_POS, yi = GENGA_SENTINEL_POS, zi = GENGA_SENTINEL_POS;
    int fi = -1, wfw = -1;
    float4 wlo = make_float4(3.0e38f, 3.0e38f, 3.0e38f, 0.0f), whi = make_float4(-3.0e38f, -3.0e38f, -3.0e38f, 0.0f);
    if (r < i_rec_end) {
        const double2 a = p.rxy[r], b = p.rzm[r];
        xi = a.x; yi = a.y; zi = b.x;
        fi = p.rfw[r];
        wlo = p.cblo[ig]; whi = p.cbhi[ig];
        wfw = __float_as_int(wlo.w);
    }
    const bool active = wfw >= 0;                           // the group holds at least one real body
    // Level >= 1 search, massive i-group against the massive j-groups: the trip rule is symmetric, so each unordered
    // pair is queued ONCE, as a symmetric candidate (half the search, half the exact path's atomics).  The particles'
    // groups and the fallback after an overflow keep ordered pairs.
    const bool sym_i = !RESCAN && !force_only && j_group0 == 0 && ig < n_jgroups;
    CandCursor cc;
    cc.base = 0;
    cc.fill = GENGA_CAND_BLOCK;
    cc.over = false;

    const int js = gridDim.y, jy = blockIdx.y;               // this CTA's j-groups: g = q * js + jy
    const int n_mine = (n_jgroups - jy + js - 1) / js;
    for (int g0 = 0; g0 < n_mine; g0 += GENGA_NEAR_BOXES) {
        __syncthreads();
        for (int q = tid; q < GENGA_NEAR_BOXES; q += GENGA_NEAR_THREADS) {
            const int g = (g0 + q) * js + jy;
            blo[q] = g < n_jgroups ? p.cblo[j_group0 + g] : make_float4(3.0e38f, 3.0e38f, 3.0e38f, __int_as_float(-1));
            bhi[q] = g < n_jgroups ? p.cbhi[j_group0 + g] : make_float4(-3.0e38f, -3.0e38f, -3.0e38f, 0.0f);
        }
        __syncthreads();
        if (!active) continue;
#pragma unroll 1
        for (int q0 = 0; q0 < GENGA_NEAR_BOXES; q0 += 32) {
            // (massive i-group in the level >= 1 search: every unordered massive pair once -- only the j-groups from its own on)
            const bool ahead = !sym_i || (g0 + q0 + lane) * js + jy >= ig;
            unsigned nearmask = __ballot_sync(0xffffffffu, ahead && boxes_near(wlo, whi, wfw, blo[q0 + lane], bhi[q0 + lane]));
            while (nearmask) {
                const int j0 = (j_group0 + (g0 + q0 + __ffs(nearmask) - 1) * js + jy) * GENGA_GROUP;
                nearmask &= nearmask - 1;
                const int fj_lane = p.rfw[j0 + lane];          // the pair rule of every pair loop: hi(r^2) < max(fw_i, fw_j)
                unsigned tm = 0;                            // bit u: pair (r, j0 + u) tripped the filter
#pragma unroll 8
                for (int u = 0; u < GENGA_GROUP; u++) {
                    const double2 xy = __ldg(p.rxy + j0 + u), zm = __ldg(p.rzm + j0 + u);   // same address in every lane
                    const int thr = max(fi, __shfl_sync(0xffffffffu, fj_lane, u));
                    const double dx = __dsub_rn(xy.x, xi), dy = __dsub_rn(xy.y, yi), dz = __dsub_rn(zm.x, zi);
                    const double r2 = fma(dz, dz, fma(dy, dy, __dmul_rn(dx, dx)));
                    tm |= (__double2hiint(r2) < thr ? 1u : 0u) << u;
                }
                if (sym_i && j0 == ig * GENGA_GROUP) tm &= lane < 31 ? ~0u << (lane + 1) : 0u;   // own group: j-record > i-record
                if (RESCAN) {
                    while (tm) {                            // per lane: its own tripped pairs, one after the other
                        const int jr = j0 + __ffs(tm) - 1;
                        tm &= tm - 1;
                        bool hit = false;
                        int lo = 0, hi = 0;
                        apply_candidate(p, r, force_only ? ~jr : jr, hit, lo, hi);
                        if (hit) {
                            const long long slot = atomicAdd(p.out_npairs + p.N, 1);
                            if (slot < p.capacity) reinterpret_cast<int2*>(p.out_pairs)[slot] = make_int2(lo, hi);
                        }
                    }
                } else {
                    unsigned todo = __reduce_or_sync(0xffffffffu, tm);
                    while (todo) {                          // warp-uniform: the j-records some lane tripped on
                        const int b = __ffs(todo) - 1;
                        todo &= todo - 1;
                        push_candidates(p, cc, (tm >> b) & 1u, sym_i ? ~r : r, j0 + b);      // (~i, j): both forces, once
                    }
                }
            }
        }
    }
    if (!RESCAN && cc.fill < GENGA_CAND_BLOCK) close_block(p, cc);
}

// ---------------------------------------------------------------------------------------------
// KickS (App. A): the level-L kick "applied only to the relevant bodies" -- over the
// pairs of a LIST (the encounter list of the level above, rows (i, j) in the caller's indices) instead
// of over all pairs.  One thread per listed pair evaluates it once (exact_pair: unfused IEEE, the
// definition's order) and adds the two terms, each with the bits its own side would compute
// (d -> -d, r^2 unchanged), to the bodies' fixed-point accumulators -- here indexed by BODY, the list
// kick uses no records and no internal order -- so the sums do not depend on the order of the list.
// The level-L pre-check of the listed pairs gives the level-L list (groupS: a compaction of the
// upper-level list) and the per-body counts.
// Force rules of sec. 8.1: a semi-active particle feels massive bodies only and acts on them only in
// TP 2; two particles do not interact.
// ---------------------------------------------------------------------------------------------
#define GENGA_STATUS_BAD_LIST_PAIR 16

__global__ void __launch_bounds__(256)
list_kick_kernel(const KickParams p, const double* __restrict__ pos, const double* __restrict__ mass, double G,
                 const int2* __restrict__ in_pairs, const int* __restrict__ in_n, long long in_rows, int tp2)
{
    constexpr int U = GENGA_EXACT_U;
    const long long total = min((long long)max(*in_n, 0), in_rows);
    const size_t N = (size_t)p.N;
    for (long long cbase = (long long)blockIdx.x * (256 * U); cbase < total; cbase += (long long)gridDim.x * (256 * U)) {
        bool hit[U];
        int lo[U], hi[U];
#pragma unroll
        for (int u = 0; u < U; u++) {
            const long long c = cbase + u * 256 + threadIdx.x;
            hit[u] = false; lo[u] = 0; hi[u] = 0;
            if (c >= total) continue;
            const int2 e = in_pairs[c];
            const int i = e.x, j = e.y;
            if (i < 0 || j < 0 || i >= p.N || j >= p.N || i == j) {
                atomicOr(p.status, GENGA_STATUS_BAD_LIST_PAIR);
                continue;
            }
            if (i >= p.n_massive && j >= p.n_massive) continue;          // two particles do not interact
            const double dx = __dsub_rn(pos[j], pos[i]), dy = __dsub_rn(pos[N + j], pos[N + i]),
                         dz = __dsub_rn(pos[2 * N + j], pos[2 * N + i]);
            const double gmi = __dmul_rn(G, mass[i]), gmj = __dmul_rn(G, mass[j]);
            const ExactResult r = exact_pair(p.rcrit, p.N, p.L, p.f, p.status, i, j, dx, dy, dz, gmj);
            if ((j < p.n_massive || tp2) && r.s != 0.0) {            // i feels j
                unsigned long long* acc = p.fx + i;
                fx_add(acc, p.fx_stride, __dmul_rn(r.s, dx), p.status);
                fx_add(acc + GENGA_FX_LIMBS * p.fx_stride, p.fx_stride, __dmul_rn(r.s, dy), p.status);
                fx_add(acc + 2 * GENGA_FX_LIMBS * p.fx_stride, p.fx_stride, __dmul_rn(r.s, dz), p.status);
                p.touched[i] = 1;
            }
            if ((i < p.n_massive || tp2) && r.W != 0.0 && gmi != 0.0) {   // j feels i
                const double si = __ddiv_rn(__dmul_rn(gmi, r.W), r.r3);
                unsigned long long* acc = p.fx + j;
                fx_add(acc, p.fx_stride, -__dmul_rn(si, dx), p.status);
                fx_add(acc + GENGA_FX_LIMBS * p.fx_stride, p.fx_stride, -__dmul_rn(si, dy), p.status);
                fx_add(acc + 2 * GENGA_FX_LIMBS * p.fx_stride, p.fx_stride, -__dmul_rn(si, dz), p.status);
                p.touched[j] = 1;
            }
            if (r.enc) {
                atomicAdd(p.out_npairs + i, 1);
                atomicAdd(p.out_npairs + j, 1);
                hit[u] = true; lo[u] = min(i, j); hi[u] = max(i, j);
            }
        }
        emit_pairs_cta<U>(p, hit, lo, hi);
    }
}

__global__ void __launch_bounds__(256)
list_reduce_kernel(unsigned long long* __restrict__ fx, long long fx_stride, int* __restrict__ touched, int N, double dt,
                   int* __restrict__ status, double* __restrict__ out_acc, double* __restrict__ vel)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= N) return;
    double a0 = 0.0, a1 = 0.0, a2 = 0.0;
    if (touched[b]) {
        touched[b] = 0;
        unsigned long long* acc = fx + b;
        a0 = fx_take(acc, fx_stride, status);
        a1 = fx_take(acc + GENGA_FX_LIMBS * fx_stride, fx_stride, status);
        a2 = fx_take(acc + 2 * GENGA_FX_LIMBS * fx_stride, fx_stride, status);
    }
    if (out_acc) {
        out_acc[b] = a0;
        out_acc[(size_t)N + b] = a1;
        out_acc[2 * (size_t)N + b] = a2;
    }
    if (vel) {
        vel[b] = fma(dt, a0, vel[b]);
        vel[(size_t)N + b] = fma(dt, a1, vel[(size_t)N + b]);
        vel[2 * (size_t)N + b] = fma(dt, a2, vel[2 * (size_t)N + b]);
    }
}

// genga_kick_merged: the candidate list was built for critical radii up to `scale` times the old ones
#define GENGA_STATUS_RCRIT_JUMP 256
__global__ void __launch_bounds__(256)
rcrit_jump_kernel(const double* __restrict__ rc_old, const double* __restrict__ rc_new, int N, double scale,
                  int* __restrict__ status)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b < N && rc_new[b] > __dmul_rn(rc_old[b], scale)) atomicOr(status, GENGA_STATUS_RCRIT_JUMP);
}

// ---------------------------------------------------------------------------------------------
// reduce_kernel (row a8 + a7): record r adds, in a FIXED order, what the pair loops
// left for it: the partial segments of its i-block in ascending CTA order (up to three pair-loop
// passes, each with its own plan), the reaction sums of the symmetric pass in ascending row order,
// and the exact path's fixed-point sum; then writes the caller's arrays.
// ---------------------------------------------------------------------------------------------
struct SegPlan {                       // the partial segments one pair-loop pass has written
    const double* __restrict__ partial;   // [n_ctas][max_segs][3][IB]
    int IB, n_j_tiles, n_ctas, max_segs;  // n_ctas == 0: the pass did not run
    long long n_tiles;
    int rec0, rec_end;                 // the pass served the i-records [rec0, rec_end), i-block 0 at rec0
    int symmetric, r, n_rows;          // kick_sym_kernel's row-major triangular tile numbering (genga_kick_variants.h)
    const long long* __restrict__ tbegin;  // symmetric: [n_ctas + 1] first tile of every CTA; else nullptr (c T / C)
};

struct ReduceParams {
    SegPlan seg[3];                    // added in this order
    const double* __restrict__ react;  // symmetric pass: [n_tiles][3][JT] reaction sums (nullptr: none); plan = seg[0]
    int react_jt;                      // its j-tile
};

__device__ __forceinline__ void add_segments(const SegPlan& q, int r, double& a0, double& a1, double& a2)
{
    if (q.n_ctas <= 0 || r < q.rec0 || r >= q.rec_end) return;
    const int ib = (r - q.rec0) / q.IB, off = (r - q.rec0) - ib * q.IB;
    const long long ta = q.symmetric ? sym_row_begin(ib, q.n_j_tiles, q.r) : (long long)ib * q.n_j_tiles;
    const long long tb = (q.symmetric ? sym_row_begin(ib + 1, q.n_j_tiles, q.r) : ta + q.n_j_tiles) - 1;
    if (tb < ta) return;
    int c_first, c_last;
    if (q.tbegin) {                                        // the largest c with tbegin[c] <= t (empty ranges repeat a value)
        auto owner = [&](long long t) {
            int lo = 0, hi = q.n_ctas - 1;
            while (lo < hi) {
                const int mid = (lo + hi + 1) >> 1;
                if (q.tbegin[mid] <= t) lo = mid; else hi = mid - 1;
            }
            return lo;
        };
        c_first = owner(ta); c_last = owner(tb);
    } else {
        c_first = plan_tile_owner(ta, q.n_tiles, q.n_ctas); c_last = plan_tile_owner(tb, q.n_tiles, q.n_ctas);
    }
    for (int c = c_first; c <= c_last; c++) {
        const long long tc = q.tbegin ? q.tbegin[c] : plan_tile_begin(c, q.n_tiles, q.n_ctas);
        if (q.tbegin && q.tbegin[c + 1] <= tc) continue;   // a CTA without tiles wrote nothing
        const int seg = ib - (q.symmetric ? sym_row_of(tc, q.n_j_tiles, q.r, q.n_rows) : (int)(tc / q.n_j_tiles));
        const double* v = q.partial + ((size_t)c * q.max_segs + seg) * 3 * q.IB + off;
        a0 = __dadd_rn(a0, v[0]);
        a1 = __dadd_rn(a1, v[q.IB]);
        a2 = __dadd_rn(a2, v[2 * (size_t)q.IB]);
    }
}

#define GENGA_REDUCE_THREADS 64      // small CTAs: 65,536 records spread evenly over 148 SMs
__global__ void __launch_bounds__(GENGA_REDUCE_THREADS)
reduce_kernel(const ReduceParams rp, const int* __restrict__ ridx, int n_rec, int N, double dt,
              unsigned long long* __restrict__ fx, long long fx_stride, int* __restrict__ touched, int* __restrict__ status,
              double* __restrict__ out_acc, double* __restrict__ vel)
{
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n_rec) return;
    const int b = ridx[r];
    if (b < 0) return;
    double a0 = 0.0, a1 = 0.0, a2 = 0.0;
    add_segments(rp.seg[0], r, a0, a1, a2);
    if (rp.react && r < rp.seg[0].rec_end) {
        // the reaction sums of the symmetric tiles that hold record r as a j-record: rows 0 .. (row of r) - 1
        const SegPlan& q = rp.seg[0];
        const int JT = rp.react_jt, jt = r / JT, off = r - jt * JT, rows = r / q.IB;
        // (loads of 8 rows in flight, added in row order)
        for (int I0 = 0; I0 < rows; I0 += 8) {
            double v0[8], v1[8], v2[8];
#pragma unroll
            for (int u = 0; u < 8; u++) {
                const int I = min(I0 + u, rows - 1);
                const long long t = sym_row_begin(I, q.n_j_tiles, q.r) + (jt - I * q.r);
                const double* v = rp.react + (size_t)t * (3 * JT) + off;
                v0[u] = v[0]; v1[u] = v[JT]; v2[u] = v[2 * JT];
            }
#pragma unroll
            for (int u = 0; u < 8; u++)
                if (I0 + u < rows) {
                    a0 = __dadd_rn(a0, v0[u]);
                    a1 = __dadd_rn(a1, v1[u]);
                    a2 = __dadd_rn(a2, v2[u]);
                }
        }
    }
    add_segments(rp.seg[1], r, a0, a1, a2);
    add_segments(rp.seg[2], r, a0, a1, a2);
    if (touched[r]) {                                      // the exact path's terms (fixed point, see fx_add)
        touched[r] = 0;
        unsigned long long* acc = fx + r;
        a0 = __dadd_rn(a0, fx_take(acc, fx_stride, status));
        a1 = __dadd_rn(a1, fx_take(acc + GENGA_FX_LIMBS * fx_stride, fx_stride, status));
        a2 = __dadd_rn(a2, fx_take(acc + 2 * GENGA_FX_LIMBS * fx_stride, fx_stride, status));
    }
    if (out_acc) {
        out_acc[b] = a0;
        out_acc[(size_t)N + b] = a1;
        out_acc[2 * (size_t)N + b] = a2;
    }
    if (vel) {
        vel[b] = fma(dt, a0, vel[b]);
        vel[(size_t)N + b] = fma(dt, a1, vel[(size_t)N + b]);
        vel[2 * (size_t)N + b] = fma(dt, a2, vel[2 * (size_t)N + b]);
    }
}

}  // namespace genga
