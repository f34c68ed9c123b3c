// WCSPH acceleration, eq.8-9 (L128-132; Listing 4):
//     a_i = g - sum_j m_j (p_i/rho_i^2 + p_j/rho_j^2 + Pi_ij) grad_i W_ij
// with Monaghan artificial viscosity Pi_ij (R9; the paper only names "the classic scheme", L185)
// and, in the same pair loop ("no inter-dependencies and may be computed together", L337), the continuity
// right-hand side eq.7 (L126; Listing 4):   arho_i = sum_j m_j (v_i - v_j) . grad_i W_ij.
// Gravity is the initial value of the accumulator (Listing 4).
#include "sph_tile.cuh"

template <int KERNEL, int DIM, bool VARH, bool PER, bool ARHO, bool FILTER>
struct AccelPolicy : QueuePolicy<AccelPolicy<KERNEL, DIM, VARH, PER, ARHO, FILTER>, FILTER, false> {
    const float4* posh; const float4* velm; const float2* rp;
    float4 pi, vi; float rho_i, pr_i;
    float ax, ay, az, ar;
    float Lx, Ly, Lz, iLx, iLy, iLz;
    float sigma, h_c, hinv_c, fac_c, visc, eps;

    __device__ __forceinline__ void body(uint32_t j) {
        const float4 pj = __ldg(posh + j);
        const float4 vj = __ldg(velm + j);
        const float2 rj = __ldg(rp + j);
        const float dx = min_image<PER>(pi.x - pj.x, Lx, iLx);
        const float dy = min_image<PER>(pi.y - pj.y, Ly, iLy);
        float dz = 0.0f;
        float r2 = fmaf(dy, dy, dx * dx);
        if (DIM == 3) { dz = min_image<PER>(pi.z - pj.z, Lz, iLz); r2 = fmaf(dz, dz, r2); }
        const float rinv = r2 > 0.0f ? rsqrt_approx(r2) : 0.0f;       // grad W := 0 at r = 0 (R18): rinv = 0
        const float r = r2 * rinv;
        float hij, hinv, fac;
        if (VARH) {
            hij = 0.5f * (pi.w + pj.w);
            hinv = rcp_approx(hij);
            fac = sigma * hinv * hinv * (DIM == 3 ? hinv : 1.0f);
        } else { hij = h_c; hinv = hinv_c; fac = fac_c; }
        float f, df;
        kernel_profile<KERNEL, DIM>(r * hinv, f, df);
        const float gc = fac * hinv * df * rinv;                        // grad_i W_ij = gc * (dx,dy,dz)
        const float vx = vi.x - vj.x, vy = vi.y - vj.y;
        float vr = fmaf(vy, dy, vx * dx);
        if (DIM == 3) vr = fmaf(vi.z - vj.z, dz, vr);
        // Pi_ij = -alpha c0 mu / rhobar, mu = h vr/(r^2 + eps h^2), rhobar = (rho_i+rho_j)/2, only if vr < 0
        const float den = fmaf(eps * hij, hij, r2) * (rho_i + rj.x);
        const float Pi = vr < 0.0f ? visc * hij * vr * rcp_approx(den) : 0.0f;
        const float s = -vj.w * gc * (pr_i + rj.y + Pi);
        ax = fmaf(s, dx, ax); ay = fmaf(s, dy, ay);
        if (DIM == 3) az = fmaf(s, dz, az);
        if (ARHO) ar = fmaf(vj.w * gc, vr, ar);
    }
};

// ARHO_ONLY launches serve ContinuityEquation(dest=solid, sources=[fluid]) (Listing 3): the same
// loop, only arho is stored.
template <class Pol>
__device__ __forceinline__ void accel_setup(Pol& pol, const GridDesc& g, const PairConsts& pc, const SortedState& S,
                                            float4 pi, float4 vi, float2 ri) {
    pol.posh = S.posh; pol.velm = S.velm; pol.rp = S.rp;
    pol.pi = pi; pol.vi = vi; pol.rho_i = ri.x; pol.pr_i = ri.y;
    pol.ax = pc.g[0]; pol.ay = pc.g[1]; pol.az = pc.g[2]; pol.ar = 0.0f;
    pol.Lx = g.L[0]; pol.Ly = g.L[1]; pol.Lz = g.L[2];
    pol.iLx = 1.0f / g.L[0]; pol.iLy = 1.0f / g.L[1]; pol.iLz = 1.0f / g.L[2];
    pol.sigma = pc.sigma; pol.h_c = pc.h_const; pol.hinv_c = pc.hinv_const; pol.fac_c = pc.fac_const;
    pol.visc = pc.visc; pol.eps = pc.eps;
}

template <int DIM, bool ARHO, class Pol>
__device__ __forceinline__ void accel_store(const Pol& pol, SortedState& S, int i, int arho_only,
                                            unsigned long long* counters) {
    float4 a = S.acc[i];
    if (arho_only) a.w = pol.ar;
    else a = make_float4(pol.ax, pol.ay, DIM == 3 ? pol.az : 0.0f, ARHO ? pol.ar : a.w);
    S.acc[i] = a;
    if (!isfinite(a.x) || !isfinite(a.y) || !isfinite(a.z) || !isfinite(a.w)) atomicAdd(&counters[CNT_NONFINITE], 1ull);
}

template <int KERNEL, int DIM, bool VARH, bool PER, bool ARHO, bool FILTER>
__global__ void __launch_bounds__(PAIR_BLOCK)
k_accel(GridDesc g, PairConsts pc, SortedState S, const uint32_t* __restrict__ cell_start, int n,
        int arho_only, unsigned long long* __restrict__ counters) {
    extern __shared__ uint32_t smem_q[];
    const int i = blockIdx.x * PAIR_BLOCK + threadIdx.x;
    const bool in = i < n;
    uint32_t meta = 0, ci = 0; float4 pi = make_float4(0, 0, 0, 1), vi = make_float4(0, 0, 0, 0);
    float2 ri = make_float2(1, 0);
    if (in) { meta = S.meta[i]; ci = S.cell[i]; pi = S.posh[i]; vi = S.velm[i]; ri = S.rp[i]; }
    const uint32_t my_mask = in ? pc.src_mask[meta >> SPH_META_IDX_BITS] : 0u;
    const bool active = my_mask != 0u;
    if (!__any_sync(SPH_FULL_MASK, active)) return;

    AccelPolicy<KERNEL, DIM, VARH, PER, ARHO, FILTER> pol;
    pol.init(smem_q, active, S.meta, my_mask);
    accel_setup(pol, g, pc, S, pi, vi, ri);

    walk_candidates<DIM, VARH>(g, pc, S.posh, cell_start, active, pi, ci, pol);
    pol.flush();

    if (active) accel_store<DIM, ARHO>(pol, S, i, arho_only, counters);
    const unsigned long long h = warp_sum_u64(pol.hits), t = warp_sum_u64(pol.tests);
    if ((threadIdx.x & 31) == 0) { atomicAdd(&counters[CNT_PAIRS_ACCEL], h); atomicAdd(&counters[CNT_CAND_ACCEL], t); }
}

// The same pair body replayed over the neighbour rows recorded by the density pass of this evaluation
// (sph_density.cu, RECORD): no candidate tests, no queue, no shared memory.  Lane l of the warp that owns
// sorted particles [32w, 32w+32) reads word l of every row of the warp's blocks (coalesced, streaming).
#define LIST_BLOCK 128
template <int KERNEL, int DIM, bool VARH, bool PER, bool ARHO>
__global__ void __launch_bounds__(LIST_BLOCK)
k_accel_list(GridDesc g, PairConsts pc, SortedState S, int n, NList nl, unsigned long long* __restrict__ counters) {
    const int i = blockIdx.x * LIST_BLOCK + threadIdx.x;
    const int lane = threadIdx.x & 31;
    const bool in = i < n;
    uint32_t meta = 0; float4 pi = make_float4(0, 0, 0, 1), vi = make_float4(0, 0, 0, 0);
    float2 ri = make_float2(1, 0);
    if (in) { meta = S.meta[i]; pi = S.posh[i]; vi = S.velm[i]; ri = S.rp[i]; }
    const bool active = in && pc.src_mask[meta >> SPH_META_IDX_BITS] != 0u;
    if (!__any_sync(SPH_FULL_MASK, active)) return;

    AccelPolicy<KERNEL, DIM, VARH, PER, ARHO, false> pol;
    pol.init(nullptr, active, nullptr, 0u);
    accel_setup(pol, g, pc, S, pi, vi, ri);

    unsigned long long pairs = 0;
    uint32_t blk = __ldg(nl.head + (i >> 5));
    while (blk) {
        const uint32_t* hdr = nl.pool + (size_t)blk * 32;
        const uint32_t next = __ldcs(hdr), rows = __ldcs(hdr + 1);
        const uint32_t* row = hdr + 32 + lane;
        uint32_t j = rows ? __ldcs(row) : SPH_NL_NONE;
        for (uint32_t t = 0; t < rows; ++t) {
            const uint32_t jn = (t + 1 < rows) ? __ldcs(row + (size_t)(t + 1) * 32) : SPH_NL_NONE;   // prefetch
            if (active && j != SPH_NL_NONE) { pol.body(j); ++pairs; }
            j = jn;
        }
        blk = next;
    }
    if (active) accel_store<DIM, ARHO>(pol, S, i, 0, counters);
    pairs = warp_sum_u64(pairs);
    if (lane == 0) atomicAdd(&counters[CNT_PAIRS_ACCEL], pairs);
}

template <int KERNEL, int DIM>
static int launch_accel_kd(sph_ctx* c, bool filter, bool want_arho, bool arho_only, bool use_list) {
    const int n = (int)c->n_total;
    if (n == 0) return SPH_OK;
    const bool per = c->grid.per[0] || c->grid.per[1] || c->grid.per[2];
    const bool varh = c->variable_h;
    SortedState& S = c->S[c->cur];
    if (use_list) {
        const int grid = (n + LIST_BLOCK - 1) / LIST_BLOCK;
#define LL(VARH, PER, ARHO) SPH_LAUNCH(c, SPH_K_ACCEL_LIST, (k_accel_list<KERNEL, DIM, VARH, PER, ARHO>), grid, LIST_BLOCK, 0, c->grid, c->pc, S, n, c->nl, c->counters)
#define LL2(VARH, PER) do { if (want_arho) LL(VARH, PER, true); else LL(VARH, PER, false); } while (0)
        if (varh) { if (per) LL2(true, true); else LL2(true, false); }
        else      { if (per) LL2(false, true); else LL2(false, false); }
#undef LL2
#undef LL
        return SPH_OK;
    }
    const int grid = (n + PAIR_BLOCK - 1) / PAIR_BLOCK;
    const size_t smem = (size_t)PAIR_QCAP * PAIR_BLOCK * sizeof(uint32_t);
    const int ao = arho_only ? 1 : 0;
#define LA(VARH, PER, ARHO, FILTER) do { \
        auto kern = k_accel<KERNEL, DIM, VARH, PER, ARHO, FILTER>; \
        SPH_CUDA_OK(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)); \
        if (c->carveout >= 0) SPH_CUDA_OK(c, cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, c->carveout)); \
        SPH_LAUNCH(c, SPH_K_ACCEL, kern, grid, PAIR_BLOCK, smem, c->grid, c->pc, S, c->cell_start, n, ao, c->counters); } while (0)
#define LA2(VARH, PER, ARHO) do { if (filter) LA(VARH, PER, ARHO, true); else LA(VARH, PER, ARHO, false); } while (0)
#define LA3(VARH, PER) do { if (want_arho) LA2(VARH, PER, true); else LA2(VARH, PER, false); } while (0)
    if (varh) { if (per) LA3(true, true); else LA3(true, false); }
    else      { if (per) LA3(false, true); else LA3(false, false); }
#undef LA3
#undef LA2
#undef LA
    return SPH_OK;
}

// ------------------------------------------------------------------------------------------------
// Warp-tile variants (sph_tile.cuh).  k_accel_tile tests its own candidates (continuity mode, custom tables);
// k_accel_masks replays the hit masks recorded by the density pass of the same evaluation and tests nothing.
// ------------------------------------------------------------------------------------------------
struct AccelSrc { float4 pj, vj; float2 rj; uint32_t aid; };

template <int KERNEL, int DIM, bool VARH, bool ARHO, bool FILTER, bool REPLAY>
__global__ void __launch_bounds__(TILE_BLOCK, TILE_MIN_BLOCKS)
k_accel_tile(GridDesc g, PairConsts pc, SortedState S, const uint32_t* __restrict__ cell_start, int n,
             int arho_only, NList nl, unsigned long long* __restrict__ counters) {
    __shared__ TileWarpSmem smem[TILE_WARPS];
    TileWarpSmem& ws = smem[threadIdx.x >> 5];
    const int i = blockIdx.x * TILE_BLOCK + threadIdx.x;
    const int warp_id = i >> 5;
    const bool in = i < n;
    uint32_t meta = 0, ci = 0; float4 pi = make_float4(0, 0, 0, 1), vi = make_float4(0, 0, 0, 0);
    float2 ri = make_float2(1, 0);
    if (in) { meta = S.meta[i]; pi = S.posh[i]; vi = S.velm[i]; ri = S.rp[i]; if (!REPLAY) ci = S.cell[i]; }
    const uint32_t my_mask = in ? pc.src_mask[meta >> SPH_META_IDX_BITS] : 0u;
    const bool active = my_mask != 0u;
    if (!__any_sync(SPH_FULL_MASK, active)) return;

    const float Lx = g.L[0], Ly = g.L[1], Lz = g.L[2];
    const float iLx = 1.0f / g.L[0], iLy = 1.0f / g.L[1], iLz = 1.0f / g.L[2];
    const float sigma = pc.sigma, h_c = pc.h_const, hinv_c = pc.hinv_const, fac_c = pc.fac_const;
    const float visc = pc.visc, eps = pc.eps;
    const float hi = VARH ? pi.w : h_c;
    const float rho_i = ri.x, pr_i = ri.y;
    float ax = pc.g[0], ay = pc.g[1], az = pc.g[2], ar = 0.0f;      // gravity = accumulator init (Listing 4)
    unsigned long long hits = 0;
    auto load = [&](uint32_t j) {
        AccelSrc s; s.pj = __ldg(S.posh + j); s.vj = __ldg(S.velm + j); s.rj = __ldg(S.rp + j); s.aid = 0u;
        if (FILTER) s.aid = __ldg(S.meta + j) >> SPH_META_IDX_BITS;
        return s;
    };
    bool per = false;                                                   // warp-uniform: some stored batch is a periodic image
    auto compute = [&](const AccelSrc& s) {
        if (FILTER) { if (!((my_mask >> s.aid) & 1u)) return; }
        if (REPLAY) { if (!active) return; }
        float dx = pi.x - s.pj.x, dy = pi.y - s.pj.y, dz = DIM == 3 ? pi.z - s.pj.z : 0.0f;
        if (per) {
            dx = min_image<true>(dx, Lx, iLx); dy = min_image<true>(dy, Ly, iLy);
            if (DIM == 3) dz = min_image<true>(dz, Lz, iLz);
        }
        float r2 = fmaf(dy, dy, dx * dx);
        if (DIM == 3) r2 = fmaf(dz, dz, r2);
        const float rinv = r2 > 0.0f ? rsqrt_approx(r2) : 0.0f;       // grad W := 0 at r = 0 (R18): rinv = 0
        const float r = r2 * rinv;
        float hij, hinv, fac;
        if (VARH) {
            hij = 0.5f * (hi + s.pj.w);
            hinv = rcp_approx(hij);
            fac = sigma * hinv * hinv * (DIM == 3 ? hinv : 1.0f);
        } else { hij = h_c; hinv = hinv_c; fac = fac_c; }
        float f, df;
        kernel_profile<KERNEL, DIM>(r * hinv, f, df);
        const float gc = fac * hinv * df * rinv;                        // grad_i W_ij = gc * (dx,dy,dz)
        const float vx = vi.x - s.vj.x, vy = vi.y - s.vj.y;
        float vr = fmaf(vy, dy, vx * dx);
        if (DIM == 3) vr = fmaf(vi.z - s.vj.z, dz, vr);
        // Pi_ij = -alpha c0 mu / rhobar, mu = h vr/(r^2 + eps h^2), rhobar = (rho_i+rho_j)/2, only if vr < 0
        const float den = fmaf(eps * hij, hij, r2) * (rho_i + s.rj.x);
        const float Pi = vr < 0.0f ? visc * hij * vr * rcp_approx(den) : 0.0f;
        const float mg = s.vj.w * gc;
        const float sc = -mg * (pr_i + s.rj.y + Pi);
        ax = fmaf(sc, dx, ax); ay = fmaf(sc, dy, ay);
        if (DIM == 3) az = fmaf(sc, dz, az);
        if (ARHO) ar = fmaf(mg, vr, ar);
        ++hits;
    };
    auto drain = [&](uint32_t nz, bool shifted) { per = shifted; tile_drain<AccelSrc>(ws, nz, load, compute); };

    TileState st; st.reset(); st.tests = 0;
    if (REPLAY) {
        tile_replay(nl, warp_id, ws, drain);
    } else {
        const int row = in ? (int)(ci / (uint32_t)g.nc[0]) : -1;
        const int sub = in ? (int)(ci % (uint32_t)g.nc[0]) : 0;
        tile_walk<DIM, VARH>(g, pc, S.posh, cell_start, active, pi, row, sub, ws, st, [&]() { drain(st.nz, st.shifted); st.reset(); });
    }
    if (active) {
        float4 a = S.acc[i];
        if (arho_only) a.w = ar;
        else a = make_float4(ax, ay, DIM == 3 ? az : 0.0f, ARHO ? ar : a.w);
        S.acc[i] = a;
        if (!isfinite(a.x) || !isfinite(a.y) || !isfinite(a.z) || !isfinite(a.w)) atomicAdd(&counters[CNT_NONFINITE], 1ull);
    }
    const unsigned long long h = warp_sum_u64(hits), t = warp_sum_u64(st.tests);
    if ((threadIdx.x & 31) == 0) { atomicAdd(&counters[CNT_PAIRS_ACCEL], h); if (!REPLAY) atomicAdd(&counters[CNT_CAND_ACCEL], t); }
}

template <int KERNEL, int DIM>
static int launch_accel_tile_kd(sph_ctx* c, bool filter, bool want_arho, bool arho_only, bool replay) {
    const int n = (int)c->n_total;
    if (n == 0) return SPH_OK;
    const bool varh = c->variable_h;
    SortedState& S = c->S[c->cur];
    const int grid = (n + TILE_BLOCK - 1) / TILE_BLOCK;
    const int ao = arho_only ? 1 : 0;
#define LT(VARH, ARHO, FILTER, REPLAY) \
        SPH_LAUNCH(c, (REPLAY ? SPH_K_ACCEL_LIST : SPH_K_ACCEL), (k_accel_tile<KERNEL, DIM, VARH, ARHO, FILTER, REPLAY>), grid, TILE_BLOCK, 0, c->grid, c->pc, S, c->cell_start, n, ao, c->nl, c->counters)
#define LT1(VARH, ARHO, FILTER) do { if (replay) LT(VARH, ARHO, FILTER, true); else LT(VARH, ARHO, FILTER, false); } while (0)
#define LT2(VARH, ARHO) do { if (filter) LT1(VARH, ARHO, true); else LT1(VARH, ARHO, false); } while (0)
#define LT3(VARH) do { if (want_arho) LT2(VARH, true); else LT2(VARH, false); } while (0)
    if (varh) LT3(true); else LT3(false);
#undef LT3
#undef LT2
#undef LT1
#undef LT
    return SPH_OK;
}

int launch_accel(sph_ctx* c, const uint32_t* src_mask_per_dest, bool want_arho, bool arho_only) {
    bool filter = false, use_list = c->nl_valid && !arho_only;
    for (int a = 0; a < SPH_MAX_ARRAYS; ++a) {
        c->pc.src_mask[a] = a < c->na ? src_mask_per_dest[a] : 0u;
        if (c->pc.src_mask[a] && c->pc.src_mask[a] != c->pc.all_mask) filter = true;
        if (c->pc.src_mask[a] && c->pc.src_mask[a] != c->nl_mask[a]) use_list = false;   // rows recorded with another mask
    }
    c->last_used_rows = use_list;
    const int k = c->prm.kernel, d = c->grid.dim;
#define KD(K, D) if (k == K && d == D) return c->tile ? launch_accel_tile_kd<K, D>(c, filter, want_arho || arho_only, arho_only, use_list) \
                                               : launch_accel_kd<K, D>(c, filter, want_arho || arho_only, arho_only, use_list)
    KD(SPH_KERNEL_CUBIC, 2); KD(SPH_KERNEL_CUBIC, 3);
    KD(SPH_KERNEL_QUINTIC, 2); KD(SPH_KERNEL_QUINTIC, 3);
    KD(SPH_KERNEL_WENDLAND_C2, 2); KD(SPH_KERNEL_WENDLAND_C2, 3);
#undef KD
    return sph_fail(c, SPH_ERR_BAD_ARG, "unsupported kernel/dim");
}
