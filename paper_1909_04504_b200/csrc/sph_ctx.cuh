// The opaque context behind sph_ctx* (library-owned; see include/sph.h "ownership").
#pragma once
#include "sph_internal.cuh"
#include <stdio.h>

// device counters: [2..5] are cleared by every evaluation / pair call, [6..8] by every search
enum { CNT_OUT_OF_DOMAIN = 0, CNT_NONFINITE = 1, CNT_PAIRS_DENSITY = 2, CNT_CAND_DENSITY = 3, CNT_PAIRS_ACCEL = 4,
       CNT_CAND_ACCEL = 5, CNT_OVERFLOW = 6, CNT_NL_USED = 7 /* low 32 bits: record rows handed out (NList::used) */,
       CNT_CAND_SEARCH = 8, CNT_ASSERT = SPH_CNT_ASSERT /* failed device-side bounds assertions (-DSPH_DEBUG_ASSERT builds) */, CNT_COUNT = 10 };

struct sph_ctx {
    cudaStream_t stream;
    int device, sm_count;
    sph_params prm;
    sph_domain dom;
    int na;
    int64_t cap[SPH_MAX_ARRAYS], cap_total;
    int64_t n[SPH_MAX_ARRAYS], base[SPH_MAX_ARRAYS + 1], n_total;   // base = offsets in concatenated caller order
    int fixed[SPH_MAX_ARRAYS];
    uint32_t tbl_density[SPH_MAX_ARRAYS], tbl_accel[SPH_MAX_ARRAYS], tbl_arho[SPH_MAX_ARRAYS];
    bool tables_user;

    GridDesc grid;
    PairConsts pc;
    bool built, have_accel, have_arho, variable_h;
    bool p_is_eos;             // every p of the state is the EOS of its rho (no array supplied p at the last build)
    real h_min, h_max;
    int64_t n_keys, max_keys;

    SortedState S[2];          // double-buffered (permute A -> B); acc is permuted only by sph_nnps_build (inside
                               // sph_pc_step it is consumed by k_update before the sort and rewritten after it)
    int cur;
    uint32_t *key, *rank;      // per particle, pre-sort order
    uint32_t *cell_count, *cell_start;
    unsigned long long* scan_state; uint32_t* scan_ticket;   // k_scan look-back table; scan_ticket[0] = ticket, [1] = epoch
    uint32_t* scan_tiles; int scan_tiles_cap;                // two-level scan of large tables: tile sums [cap + 1] and tile prefixes [cap + 1]
    real* staging;             // host<->device staging for SPH_MEM_HOST (14 reals per particle of capacity)
    unsigned long long* counters;     // device, CNT_COUNT entries
    void* hminmax;             // device, 4 x 8 bytes: h min/max, |m| min/max as ordered integers of the real type

    // neighbour rows recorded by a density launch for the acceleration launch that follows it
    NList nl;                  // nl.pool == nullptr: recording disabled
    bool nl_valid;             // the records match the current sorted order (launch_search ran since the last sort)
    bool inv_valid;            // rank[] holds the inverse permutation (caller order -> sorted index) of the current order
    bool last_used_rows;       // the last acceleration launch replayed recorded rows
    bool counters_fresh;       // k_update has just cleared the counters of the search and the pair passes (consumed by evaluate)
    bool heads_fresh;          // k_scatter has just cleared the record heads (consumed by launch_search)
    // CUDA graph of two consecutive steps of sph_pc_step (the state buffers flip every step), replayed for long runs
    cudaGraphExec_t step_graph; real graph_dt; int graph_cont, graph_cur, graph_nodes; bool graph_off;
    int xsub;                  // x sub-cells per support radius requested (GridDesc::xsub is what the grid got)

    int64_t launches, steps_done;
    // profiling: event pairs around launches (sph_set_profiling)
    bool prof_on;
    struct ProfRec { cudaEvent_t a, b; int id; }* prof;
    int prof_cap, prof_used; int64_t prof_dropped;
    int64_t last_pairs_density, last_pairs_accel;
    char err[512];
};

#define SPH_CUDA_OK(ctx, expr) do { cudaError_t e__ = (expr); if (e__ != cudaSuccess) { \
    snprintf((ctx)->err, sizeof((ctx)->err), "%s: %s (%s:%d)", #expr, cudaGetErrorString(e__), __FILE__, __LINE__); \
    return SPH_ERR_CUDA; } } while (0)

static inline int sph_fail(sph_ctx* c, int code, const char* msg) {
    if (c) snprintf(c->err, sizeof(c->err), "%s", msg);
    return code;
}

// launch accounting: every kernel of the library goes through this macro
int sph_prof_begin(sph_ctx* c, int id);          // returns the record index or -1
void sph_prof_end(sph_ctx* c, int rec);
#define SPH_LAUNCH(ctx, kid, kernel, grid, block, smem, ...) do { \
    const int rec__ = (ctx)->prof_on ? sph_prof_begin((ctx), (kid)) : -1; \
    kernel<<<(grid), (block), (smem), (ctx)->stream>>>(__VA_ARGS__); (ctx)->launches++; \
    if (rec__ >= 0) sph_prof_end((ctx), rec__); \
    cudaError_t e__ = cudaPeekAtLastError(); if (e__ != cudaSuccess) { \
        snprintf((ctx)->err, sizeof((ctx)->err), "launch %s: %s", #kernel, cudaGetErrorString(e__)); \
        return SPH_ERR_CUDA; } } while (0)

struct PackSrc { const real *x, *y, *z, *u, *v, *w, *h, *m, *rho, *p, *ax, *ay, *az, *arho; };
struct PackArgs { PackSrc a[SPH_MAX_ARRAYS]; long long base[SPH_MAX_ARRAYS + 1]; int na; };
struct OutPtrs { real *x, *y, *z, *u, *v, *w, *rho, *p, *ax, *ay, *az, *arho; };

// sph_nnps.cu
int nnps_pack(sph_ctx* c, const PackArgs& A);        // caller SoA -> float4 groups (unsorted) + h_min/h_max
int nnps_key_hist(sph_ctx* c);                       // key + rank + histogram from S[cur]
int nnps_update_key_hist(sph_ctx* c, real dt, bool kick2, bool kick1_drift, bool continuity, bool rekey);
int nnps_sort_from_keys(sph_ctx* c, bool with_acc);  // scan + scatter (key/rank/cell_count filled); swaps buffers
int nnps_gather_out(sph_ctx* c, int array, const OutPtrs& O);
int nnps_stencil_candidates(sph_ctx* c, int64_t* out);
int nnps_export_neighbors(sph_ctx* c, int dest, int src, int64_t* offsets, int32_t* indices, int64_t cap,
                          int64_t* total, int mem);
// sph_density.cu / sph_accel.cu: one launch serves every dest array whose mask is non-zero
int launch_search(sph_ctx* c);                       // sph_search.cu: records the candidate masks of the current sorted order
int launch_density(sph_ctx* c, const uint32_t* src_mask_per_dest);
// what a momentum launch stores for which array (bitmasks over arrays)
struct AccelRoles {
    uint32_t arho_only;        // destination arrays that store only their continuity sum (acc.w)
    uint32_t keep_xyz;         // ... of those, arrays whose acc.xyz an earlier launch of this evaluation computed (kept); the others get 0
    uint32_t zero_xyz, zero_w; // arrays that are NO destination of this launch and whose acc.xyz / acc.w no launch of the evaluation computes: zeroed
};
int launch_accel(sph_ctx* c, const uint32_t* src_mask_per_dest, bool want_arho, const AccelRoles& roles);
