// Neighbour search of one sorted order (Sec.2.2), run ONCE per rebuild of the NNPS and shared by
// every pair pass of the evaluation (summation density, momentum, continuity): the warp-tile walker of sph_tile.cuh
// streams the candidate runs of every group through the tensor-core filter and writes the candidate masks, bases and
// shift codes to the record pool.  The pair kernels replay the records and apply the exact predicate (R7)
// and their own source-array masks; the paper's own diagnosis of its 2x gap to DualSPHysics is the separate
// neighbour pass per equation group (L750) -- here every group of an evaluation reuses one search.
#include "sph_tile.cuh"

template <int DIM, bool VARH>
__global__ void __launch_bounds__(TILE_BLOCK, TILE_MIN_BLOCKS)
k_search_tile(GridDesc g, PairConsts pc, SortedState S, const uint32_t* __restrict__ cell_start, int n,
              NList nl, unsigned long long* __restrict__ counters) {
    typedef TileWarpSmemT<TILE_MMAX_OF(VARH)> WS;
    __shared__ WS smem[TILE_WARPS];
    WS& ws = smem[threadIdx.x >> 5];
    const int i = blockIdx.x * TILE_BLOCK + threadIdx.x;
    const int warp_id = i >> 5;
    const bool in = i < n;
    uint32_t ci = 0; float4 pi = make_float4(0, 0, 0, 1);
    if (in) { ci = S.cell[i]; pi = to_float4(ldg_r(S.posh + i)); }
    TileState st; st.reset(); st.tests = 0;
    TileRecorder rec; rec.init(nl);
    tile_walk<DIM, VARH>(g, pc, S.posh, cell_start, in, in, pi, ci, ws, st,
                         [&]() { rec.append(ws, st.M, st.shifted, warp_id, counters); st.reset(); });
    const unsigned long long t = warp_sum_u64((unsigned long long)st.tests);
    if ((threadIdx.x & 31) == 0) atomicAdd(&counters[CNT_CAND_SEARCH], t);
}

// Records the candidate masks of the current sorted order for every particle (all arrays as destinations and as
// sources).  Needs the record pool; the pair launches that follow replay it until the next sort.
int launch_search(sph_ctx* c) {
    c->nl_valid = false;
    const int n = (int)c->n_total;
    if (c->nl.pool == nullptr || n == 0) return SPH_OK;
    if (!c->heads_fresh)           // (inside sph_pc_step k_scatter and k_update have already cleared both)
        SPH_CUDA_OK(c, cudaMemsetAsync(c->nl.head, 0, (size_t)((c->n_total + 31) / 32 + 1) * sizeof(uint32_t), c->stream));
    if (!c->counters_fresh)
        SPH_CUDA_OK(c, cudaMemsetAsync(c->counters + CNT_OVERFLOW, 0, (size_t)(CNT_CAND_SEARCH - CNT_OVERFLOW + 1) * sizeof(unsigned long long), c->stream));
    c->heads_fresh = false;
    const int grid = (n + TILE_BLOCK - 1) / TILE_BLOCK;
    SortedState& S = c->S[c->cur];
#define LS(DIM, VARH) SPH_LAUNCH(c, SPH_K_SEARCH, (k_search_tile<DIM, VARH>), grid, TILE_BLOCK, 0, c->grid, c->pc, S, c->cell_start, n, c->nl, c->counters)
    if (c->grid.dim == 2) { if (c->variable_h) LS(2, true); else LS(2, false); }
    else                  { if (c->variable_h) LS(3, true); else LS(3, false); }
#undef LS
    c->nl_valid = true;
    return SPH_OK;
}
