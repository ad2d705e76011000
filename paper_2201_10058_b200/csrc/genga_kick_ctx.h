// The context of the C-ABI library (include/genga_kick.h, include/genga_step.h): private to csrc/.
#pragma once
#include "../../include/genga_kick.h"
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>

struct genga_kick_ctx {
    genga_kick_config cfg;
    int64_t N;
    int num_sms;
    cudaStream_t stream;
    genga_kick_plan* plans;        // one per level 0..max_level
    genga_kick_plan plan_tp2;      // TP 2: second pass of the level-0 kick (massive i x semi-active j)
    bool tp2;
    double* partial2;              // its partial sums
    genga_kick_plan plan_sym;      // level 0, massive x massive, every unordered pair once (n_ctas == 0: not used)
    genga_kick_plan plan_tprows;   // ... and the one-sided rows of the semi-active particles beside it
    double* partial_sym;           // i-side partial sums of the symmetric pass
    double* react;                 // its reaction sums, one slot per tile
    long long* sym_t0;             // [n_ctas + 1] first tile of every CTA of the symmetric pass (device)
    // scratch (device)
    double2* rxy;
    double2* rzm;
    int* rfw;
    int* ridx;
    float4* cblo;
    float4* cbhi;
    // internal order (genga_kick_sort.cuh); sorted == false: caller's order
    bool sorted;
    bool reuse_order;              // genga_kick_set_order_reuse: keep the permutation of the last sort
    bool order_valid;              // ... there is one
    bool reuse_list;               // genga_kick_set_order_reuse(2): level >= 1 kicks also take the candidate list of the
                                   // last level-0 kick (positions unchanged since then)
    bool list_valid;               // ... ctx->cand holds one (the last kick that wrote a list was a level-0 kick)
    int* rfw_ref;                  // [n_rec] filter words that list was built with
    int* need_near;                // [max_level + 1] != 0: some body's filter word at that level exceeds rfw_ref
    int sort_blocks;
    unsigned* bbox;
    unsigned* keys_a;
    unsigned* keys_b;
    int* vals_a;                   // ends up holding the permutation
    int* vals_b;
    int* counts;
    double* partial;
    int* status;
    // exact path: candidate list, fixed-point accumulators (genga_kick_kernels.cuh)
    int2* cand;
    int64_t cand_capacity;
    int* ncand;
    unsigned long long* fx;
    int* touched;
    int64_t n_rec_alloc;
    // staging for genga_kick_host (device, lazily allocated)
    double* h_pos; double* h_vel; double* h_mass; double* h_rcrit; double* h_acc;
    int32_t* h_pairs; int32_t* h_npairs;
    int64_t launches;
    // measurement aids (genga_kick_enable_timing)
    bool timing;
    cudaEvent_t* ev;               // [max_level + 1][2], created by genga_kick_enable_timing
    bool* ev_set;                  // [max_level + 1]
    // O(N) neighbours of the kick (genga_step.cu), lazily allocated
    double* psum_partial;          // [GENGA_PSUM_BLOCKS][3] block sums of m v, then the totals at [GENGA_PSUM_BLOCKS][3]
    unsigned* psum_ticket;         // last-block-done counter, zero between launches
    double* step_rcrit;            // [N] row Rcrit(dt) of genga_step when the caller keeps none
    // grouping (genga_group.cu), lazily allocated
    int* grp_label; int* grp_flag; unsigned* grp_keys_a; unsigned* grp_keys_b; int* grp_vals_a; int* grp_vals_b;
    int* grp_counts;
    double* bs_scratch;            // whole-grid Bulirsch-Stoer regime: positions (2 buffers), G m, r_crit rows, error slots
    int32_t* bs_stats;             // caller's per-group record of the step-size control, or nullptr (genga_bs_set_stats)
    int64_t bs_stats_rows;
    int* bs_nbr;                   // ... neighbour lists of the group being integrated
    long long bs_nbr_capacity;
    int bs_coop_blocks;            // its co-resident grid (eight lanes per body)
    int bs_coop_blocks1;           // ... of the one-lane-per-body variant
    int bs_coop_blocks_by_lanes[4];// co-resident grids of the variants with 8, 4, 2, 1 lanes per body
    int bs_teams;                  // teams of GENGA_BS_TEAM_CTAS CTAs that grid is cut into
    long long bs_rows;             // rows of every array of bs_scratch
    double* hyb_state;             // [6][N] state before FG (genga_hybrid_step), lazily allocated
    void* senc_slab;               // scratch of genga_multilevel_step (genga_senc.cu), lazily allocated
    int senc_levels;               // levels it was cut for
    std::string cuda_err;
};


static inline int genga_cuda_fail(genga_kick_ctx* ctx, cudaError_t e)
{
    if (ctx) ctx->cuda_err = cudaGetErrorString(e);
    return GENGA_KICK_E_CUDA;
}
#define GK_CUDA(ctx, call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return genga_cuda_fail(ctx, e_); } while (0)

static inline bool genga_misaligned(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) != 0; }

// genga_kick with out_npairs == nullptr allowed: no pre-check output (the closing kick of genga_step)
int genga_kick_impl(genga_kick_ctx* ctx, const double* pos, double* vel, const double* mass, const double* rcrit,
                    int32_t changeover_level, double dt, double* out_acc, int32_t* out_pairs, int32_t* out_npairs);
// genga_group with a status bit to raise when the pair list was clipped to pair_rows (0: none, the public call)
int genga_group_impl(genga_kick_ctx* ctx, const int32_t* pairs, const int32_t* n_pairs, int64_t pair_rows,
                     int32_t* group_of, int32_t* members, int32_t* offsets, int32_t* summary, int clip_status);
// closing Kick(dt_step / 2) of a step + Rcrit(dt_step) + opening Kick(dt_step / 2) with pre-check of the next, in one
// pass over the pairs (genga_kick.cu); rc_old: the row of the step that ends, rc_new: [N] receives the next step's row
int genga_kick_merged_impl(genga_kick_ctx* ctx, const double* pos, double* vel, const double* mass, const double* rc_old,
                           double* rc_new, double m_star, double dt_step, double n1, double n2, double* out_acc,
                           int32_t* out_pairs, int32_t* out_npairs);
