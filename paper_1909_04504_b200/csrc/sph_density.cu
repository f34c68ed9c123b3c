// Summation density, eq.3 (L112): rho_i = sum_j m_j W(x_i - x_j, h_ij), with the Tait EOS
// (eq.6, Listing 4) fused as the epilogue (the group barrier of L337/L382 is the kernel
// boundary: every p is stored before the acceleration kernel starts).  A RECORD launch also writes the
// hit masks of its candidate tests (sph_tile.cuh), for the acceleration pass of the same evaluation to replay.
#include "sph_tile.cuh"

struct DensitySrc { float4 pj; float mj; uint32_t aid; };

template <int KERNEL, int DIM, bool VARH, bool FILTER, bool RECORD, bool UM>
__global__ void __launch_bounds__(TILE_BLOCK, TILE_MIN_BLOCKS)
k_density_tile(GridDesc g, PairConsts pc, SortedState S, const uint32_t* __restrict__ cell_start, int n,
               NList nl, unsigned long long* __restrict__ counters) {
    __shared__ TileWarpSmem smem[TILE_WARPS];
    TileWarpSmem& ws = smem[threadIdx.x >> 5];
    const int i = blockIdx.x * TILE_BLOCK + threadIdx.x;
    const int warp_id = i >> 5;
    const bool in = i < n;
    uint32_t meta = 0, ci = 0; float4 pi = make_float4(0, 0, 0, 1);
    if (in) { meta = S.meta[i]; ci = S.cell[i]; pi = S.posh[i]; }
    const uint32_t my_mask = in ? pc.src_mask[meta >> SPH_META_IDX_BITS] : 0u;
    const bool active = my_mask != 0u;
    if (!__any_sync(SPH_FULL_MASK, active)) return;
    const int row = in ? (int)(ci / (uint32_t)g.nc[0]) : -1;
    const int sub = in ? (int)(ci % (uint32_t)g.nc[0]) : 0;

    const float Lx = g.L[0], Ly = g.L[1], Lz = g.L[2];
    const float iLx = 1.0f / g.L[0], iLy = 1.0f / g.L[1], iLz = 1.0f / g.L[2];
    const float sigma = pc.sigma, hinv_c = pc.hinv_const, fac_c = pc.fac_const;
    const float hi = VARH ? pi.w : pc.h_const;
    const float mfac_c = pc.m_const * pc.fac_const;                     // UM layout: posh.w is p/rho^2, the mass is m_const
    float rho = 0.0f;
    unsigned long long fhits = 0;                                       // FILTER: hits that pass the source mask
    // constant h: posh.w of the sorted state carries the MASS (SortedState), one 16-byte gather per pair
    auto load = [&](uint32_t j) {
        DensitySrc s; s.pj = __ldg(S.posh + j); s.mj = 0.0f; s.aid = 0u;
        if (VARH) s.mj = __ldg(&S.velm[j].w);
        if (FILTER) s.aid = __ldg(S.meta + j) >> SPH_META_IDX_BITS;
        return s;
    };
    bool per = false;                                                   // warp-uniform: some stored batch is a periodic image
    auto compute = [&](const DensitySrc& s, bool has) {
        if (FILTER) { has = has && ((my_mask >> s.aid) & 1u); fhits += has ? 1u : 0u; }
        float dx = pi.x - s.pj.x, dy = pi.y - s.pj.y, dz = DIM == 3 ? pi.z - s.pj.z : 0.0f;
        if (per) {
            dx = min_image(dx, Lx, iLx); dy = min_image(dy, Ly, iLy);
            if (DIM == 3) dz = min_image(dz, Lz, iLz);
        }
        float r2 = fmaf(dy, dy, dx * dx);
        if (DIM == 3) r2 = fmaf(dz, dz, r2);
        const float rinv = r2 > 0.0f ? rsqrt_approx(r2) : 0.0f;
        const float r = r2 * rinv;
        float hinv, mfac;
        if (VARH) {
            hinv = rcp_approx(0.5f * (hi + s.pj.w));
            mfac = s.mj * sigma * hinv * hinv * (DIM == 3 ? hinv : 1.0f);
        } else { hinv = hinv_c; mfac = UM ? mfac_c : s.pj.w * fac_c; }
        float f, df;
        kernel_profile<KERNEL, DIM>(r * hinv, f, df);
        rho = has ? fmaf(mfac, f, rho) : rho;
    };

    TileState st; st.reset(); st.tests = 0; st.hits = 0;
    const uint32_t idle = in ? (uint32_t)i : 0u;
    TileRecorder rec; rec.init(nl); if (!RECORD) rec.ok = false;
    auto drain = [&]() {
        if (RECORD) rec.append(ws, st.M, st.shifted, warp_id, counters);
        per = st.shifted;
        tile_drain<DensitySrc, TILE_DRAIN_DEPTH_DENSITY>(ws, st.nz, idle, load, compute);
        st.reset();
    };
    tile_walk<DIM, VARH>(g, pc, S.posh, cell_start, active, pi, row, sub, ws, st, drain);

    if (active) {
        const float p = eos_pressure(rho, pc.rho0, pc.B, pc.gamma, pc.gamma_is_7);
        S.rp[i] = make_float2(rho, p / (rho * rho));
        // The .w stores below touch words that NO thread of this launch reads (constant h: the tests and the drain
        // use x,y,z of posh and, without UM, its .w = m, which is not written), so concurrent 16-byte gathers of the
        // same record by other warps see unchanged x,y,z whichever version of .w they get.
        if (!VARH) S.velm[i].w = rho;                                   // constant h: velm.w carries rho (SortedState)
        if (UM) S.posh[i].w = p / (rho * rho);                          // UM layout: posh.w carries p/rho^2
        if (!isfinite(rho) || !(rho > 0.0f)) atomicAdd(&counters[CNT_NONFINITE], 1ull);
    }
    const unsigned long long h = warp_sum_u64(FILTER ? fhits : st.hits), t = warp_sum_u64(st.tests);
    if ((threadIdx.x & 31) == 0) { atomicAdd(&counters[CNT_PAIRS_DENSITY], h); atomicAdd(&counters[CNT_CAND_DENSITY], t); }
}

template <int KERNEL, int DIM>
static int launch_density_tile_kd(sph_ctx* c, bool filter, bool record) {
    const int n = (int)c->n_total;
    if (n == 0) return SPH_OK;
    const int grid = (n + TILE_BLOCK - 1) / TILE_BLOCK;
    SortedState& S = c->S[c->cur];
#define LD(VARH, FILTER, RECORD, UM) \
        SPH_LAUNCH(c, SPH_K_DENSITY, (k_density_tile<KERNEL, DIM, VARH, FILTER, RECORD, UM>), grid, TILE_BLOCK, 0, c->grid, c->pc, S, c->cell_start, n, c->nl, c->counters)
#define LD2(VARH, FILTER, UM) do { if (record) LD(VARH, FILTER, true, UM); else LD(VARH, FILTER, false, UM); } while (0)
#define LD3(VARH, UM) do { if (filter) LD2(VARH, true, UM); else LD2(VARH, false, UM); } while (0)
    if (c->variable_h) LD3(true, false); else if (c->pc.uniform_m) LD3(false, true); else LD3(false, false);
#undef LD3
#undef LD2
#undef LD
    return SPH_OK;
}

// One launch computes rho,p for every array whose src_mask_per_dest entry is non-zero.
int launch_density(sph_ctx* c, const uint32_t* src_mask_per_dest, bool record) {
    bool filter = false;
    for (int a = 0; a < SPH_MAX_ARRAYS; ++a) {
        c->pc.src_mask[a] = a < c->na ? src_mask_per_dest[a] : 0u;
        if (c->pc.src_mask[a] && c->pc.src_mask[a] != c->pc.all_mask) filter = true;
    }
    record = record && c->nl.pool != nullptr && c->n_total > 0;
    c->nl_valid = false;
    if (record) {
        SPH_CUDA_OK(c, cudaMemsetAsync(c->nl.head, 0, (size_t)((c->n_total + 31) / 32 + 1) * sizeof(uint32_t), c->stream));
        // nl.used and the overflow counter live in the counter block the caller has just cleared (CNT_NL_USED)
    }
    const int k = c->prm.kernel, d = c->grid.dim;
    int rc = sph_fail(c, SPH_ERR_BAD_ARG, "unsupported kernel/dim");
#define KD(K, D) if (k == K && d == D) rc = launch_density_tile_kd<K, D>(c, filter, record)
    KD(SPH_KERNEL_CUBIC, 2); KD(SPH_KERNEL_CUBIC, 3);
    KD(SPH_KERNEL_QUINTIC, 2); KD(SPH_KERNEL_QUINTIC, 3);
    KD(SPH_KERNEL_WENDLAND_C2, 2); KD(SPH_KERNEL_WENDLAND_C2, 3);
#undef KD
    if (rc == SPH_OK && record) {
        c->nl_valid = true;
        for (int a = 0; a < SPH_MAX_ARRAYS; ++a) c->nl_mask[a] = c->pc.src_mask[a];
    }
    return rc;
}

