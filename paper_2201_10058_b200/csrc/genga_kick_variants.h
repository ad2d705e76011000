// Kernel shapes the library is compiled for, shared by the host planner (genga_kick_plan.cpp)
// and the launcher (genga_kick.cu).  A variant fixes threads per CTA, i-bodies per thread, the
// j-tile length and the CTAs per SM the kernel is bounded for (__launch_bounds__).
//
// The variants are the shapes of the level-0 pair loop (every pair contributes; 16 FP64-pipe
// instructions per pair).  changeover_level >= 1 does not use them: there W_L = 0 exactly for
// r >= rc0_ij (factor 1 - K_0 of eq. 63) and the kick is a neighbour search
// (near_kernel).
#pragma once
#include <stdint.h>

#if defined(__CUDACC__)
#define GENGA_HD __host__ __device__ __forceinline__
#else
#define GENGA_HD static inline
#endif

// Tile ranges of the decomposition (genga_kick_plan): CTA c of C owns tiles [c T / C, (c+1) T / C).
GENGA_HD long long plan_tile_begin(long long c, long long T, long long C) { return (c * T) / C; }
// The CTA that owns tile t: the largest c with floor(c T / C) <= t.
GENGA_HD int plan_tile_owner(long long t, long long T, long long C) { return (int)(((t + 1) * C - 1) / T); }

// ---- the symmetric level-0 pair loop (kick_sym_kernel): massive x massive, every unordered pair once ----
// (6 i-bodies per thread: 254 registers without spills; 8 would issue 4 % fewer instructions per pair but leaves the
// register allocator no room, and the smaller tiles balance better.)
// Rows = i-blocks of GENGA_SYM_IBLOCK records; row I holds the j-tiles jt = I r .. n_jt - 1 (r = i_block / j_tile): the
// first r of them overlap the i-block itself (the DIAGONAL tiles, evaluated one-sidedly), the others lie beyond it (the
// SYMMETRIC tiles: the force on i and the reaction on j from one evaluation).  Tiles are numbered row-major.
static const int GENGA_SYM_THREADS = 256;
static const int GENGA_SYM_IPT = 6;
static const int GENGA_SYM_JT = 256;               // = 32 x warps of the CTA (one j-group per warp and phase)
static const int GENGA_SYM_IBLOCK = GENGA_SYM_THREADS * GENGA_SYM_IPT;
static const int GENGA_SYM_MIN_BODIES = 24576;     // below this the one-sided kernel's finer tiles balance better
static const int64_t GENGA_SYM_MAX_REACT_BYTES = (int64_t)2 << 30;   // reaction partial sums: T x 3 x JT doubles
// Cost model of the static partition (CTA c owns the tiles whose cumulative cost starts in [c W / C, (c + 1) W / C)):
// a diagonal tile evaluates i_block x j_tile ORDERED pairs, most of them in the checked loop (the block's own bodies
// and their neighbours are inside each other's filter radius), a symmetric tile as many UNORDERED pairs in the bare
// loop; measured on the disks of BASELINE.json (profiles/ncu_r02*.md).
static const int GENGA_SYM_COST_SYM = 10;
static const int GENGA_SYM_COST_DIAG = 14;
// first tile of row I
GENGA_HD long long sym_row_begin(long long I, long long n_jt, long long r) { return I * n_jt - r * (I * (I - 1) / 2); }
// the row that holds tile t (rows 0 .. n_rows - 1, t < sym_row_begin(n_rows))
GENGA_HD int sym_row_of(long long t, long long n_jt, long long r, int n_rows)
{
    int lo = 0, hi = n_rows - 1;                   // largest I with sym_row_begin(I) <= t
    while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (sym_row_begin(mid, n_jt, r) <= t) lo = mid; else hi = mid - 1;
    }
    return lo;
}

struct genga_variant {
    int32_t threads;
    int32_t i_per_thread;
    int32_t j_tile;
    int32_t ctas_per_sm;
};

static const int GENGA_N_VARIANTS = 3;

// ordered from the large-N shape to the small-N shape; the planner takes the first one that
// gives every CTA at least GENGA_MIN_TILES_PER_CTA tiles, else the last
static const genga_variant GENGA_VARIANTS[GENGA_N_VARIANTS] = {
    {256, 2, 256, 2},
    {128, 2, 128, 4},
    {128, 1, 64, 4},
};
static const int GENGA_MIN_TILES_PER_CTA = 4;
static const int GENGA_NEAR_JSPLIT = 8;            // near_kernel: CTAs per i-chunk, j-groups dealt round-robin
static const int GENGA_MAX_WAVES = 4;               // CTAs launched = SMs x CTAs per SM x waves (planner)
static const int GENGA_TILES_PER_CTA_FOR_WAVES = 16; // a further wave only while every CTA keeps this many tiles
static const int GENGA_STAGES = 4;          // depth of the j-tile ring in shared memory
static const int GENGA_M_ALIGN = 256;      // every j_tile divides it
static const int GENGA_SORT_MIN_BODIES = 4096;   // GENGA_KICK_ORDER_AUTO sorts from here on
static const int GENGA_REC_ALIGN = 1024;   // every i_block divides it
// capacity of the candidate list of the exact path: pairs (ordered) inside the largest critical
// radius of either body; the mean is ~16 per body at N = 65,536
static const int64_t GENGA_CAND_PER_BODY = 64;
static const int64_t GENGA_CAND_MIN = (int64_t)1 << 20;
static const int64_t GENGA_CAND_MAX = (int64_t)1 << 28;
// genga_kick_merged: the filter radius of the shared far-field pass is that of the old critical radii times 1 + this
static const double GENGA_MERGE_MARGIN = 1.0 / 64.0;
static const int64_t GENGA_MAX_BODIES = (int64_t)1 << 30;
