// Summation density, eq.3 (L112): rho_i = sum_j m_j W(x_i - x_j, h_ij), with the Tait EOS
// (eq.6, Listing 4) fused as the epilogue (the group barrier of L337/L382 is the kernel
// boundary: every p is stored before the acceleration kernel starts).  A REPLAY launch takes its candidates from
// the records of launch_search (sph_search.cu) and walks nothing; otherwise the warp searches itself.
#include "sph_tile.cuh"

struct DensitySrc { real4 pj; real mj; uint32_t aid;
#ifdef SPH_EXP_RED
    uint32_t j;
#endif
};

template <int KERNEL, int DIM, bool VARH, bool FILTER, bool REPLAY, bool UM>
__global__ void __launch_bounds__(TILE_BLOCK, TILE_MIN_BLOCKS_DENSITY)
k_density_tile(GridDesc g, PairConsts pc, SortedState S, const uint32_t* __restrict__ cell_start, int n,
               NList nl, unsigned long long* __restrict__ counters) {
    typedef TileWarpSmemT<TILE_MMAX_OF(VARH)> WS;
    __shared__ WS smem[TILE_WARPS];
    WS& ws = smem[threadIdx.x >> 5];
    const int i = blockIdx.x * TILE_BLOCK + threadIdx.x;
    const int warp_id = i >> 5;
    const bool in = i < n;
    uint32_t meta = 0, ci = 0; real4 pi = make_real4(0, 0, 0, 1);
    if (in) { meta = S.meta[i]; ci = S.cell[i]; pi = ld_state(S.posh + i); }
    const uint32_t my_mask = in ? pc.src_mask[meta >> SPH_META_IDX_BITS] : 0u;
    const bool active = my_mask != 0u;
    if (!__any_sync(SPH_FULL_MASK, active)) return;

    const real Lx = g.Lr[0], Ly = g.Lr[1], Lz = g.Lr[2];
    const real sigma = pc.sigma, hinv_c = pc.hinv_const, fac_c = pc.fac_const;
    const real kh = sizeof(real) == 8 ? pc.ksup : pc.kh;               // what pair_cut2 of the build's real type takes
    const real hi = VARH ? pi.w : pc.h_const;
    const real cut2c = pair_cut2(kh, pc.h_const, pc.h_const);
    const real mfac_c = pc.m_const * pc.fac_const;                      // UM layout: posh.w is p/rho^2, the mass is m_const
    unsigned nhits = 0;                                                 // pairs that pass the exact predicate (and the source mask)
    // constant h: posh.w of the sorted state carries the MASS (SortedState), one 16-byte gather per pair.  Plain
    // loads: the epilogue of this launch rewrites .w words of posh / velm that other warps' gathers cover (x, y, z
    // never change and the .w they return is not used then).
    auto load = [&](uint32_t j) {
        SPH_DBG_ASSERT(j < g.n_sorted, g);
        DensitySrc s; s.pj = ld_state(S.posh + j); s.mj = 0; s.aid = 0u;
#ifdef SPH_EXP_RED
        s.j = j;
#endif
        if (VARH && !UM) s.mj = ld_state(&S.velm[j].w);            // VU layout (variable h, uniform mass): m = m_const
        if (FILTER) s.aid = __ldg(S.meta + j) >> SPH_META_IDX_BITS;
        return s;
    };
#ifdef SPH_REAL_DOUBLE
    real rho = 0.0;
    // the double build: one candidate at a time, plain double arithmetic
    auto compute = [&](const DensitySrc& s, bool has, uint32_t code, auto per) {
        real dx = rsub(pi.x, s.pj.x), dy = rsub(pi.y, s.pj.y), dz = DIM == 3 ? rsub(pi.z, s.pj.z) : real(0);
        if (decltype(per)::value) {
            dx = rsub(dx, img_shift(code, 0, Lx)); dy = rsub(dy, img_shift(code, 1, Ly));
            if (DIM == 3) dz = rsub(dz, img_shift(code, 2, Lz));
        }
        const real r2 = pair_r2(dx, dy, dz);
        has = has && r2 < (VARH ? pair_cut2(kh, hi, s.pj.w) : cut2c);
        if (FILTER) has = has && ((my_mask >> s.aid) & 1u);
        nhits += has ? 1u : 0u;
        const real r = sqrt(r2);
        real hinv, mfac;
        if (VARH) {
            hinv = real(1) / (real(0.5) * (hi + s.pj.w));
            mfac = (UM ? pc.m_const : s.mj) * sigma * hinv * hinv * (DIM == 3 ? hinv : real(1));
        } else { hinv = hinv_c; mfac = UM ? mfac_c : s.pj.w * fac_c; }
        real f, df;
        kernel_profile<KERNEL, DIM>(r * hinv, f, df);
        rho = has ? rfma(mfac, f, rho) : rho;
    };
#else
    float2 rho2 = pk1(0.0f);                                            // two partial sums: even / odd candidates of the lane
    const float2 xi2 = pk1(pi.x), yi2 = pk1(pi.y), zi2 = pk1(pi.z);
    // two candidates (a, b) of this lane at a time, packed f32x2
    auto compute = [&](const DensitySrc& a, const DensitySrc& b, bool ha, bool hb, uint32_t ca, uint32_t cb, auto per) {
        // the exact predicate of DESIGN.md R7 on the candidates the tensor-core filter let through
        float2 dx = sub2(xi2, pk(a.pj.x, b.pj.x)), dy = sub2(yi2, pk(a.pj.y, b.pj.y));
        float2 dz = DIM == 3 ? sub2(zi2, pk(a.pj.z, b.pj.z)) : pk1(0.0f);
        if (decltype(per)::value) {
            dx = sub2(dx, pk(img_shift(ca, 0, Lx), img_shift(cb, 0, Lx))); dy = sub2(dy, pk(img_shift(ca, 1, Ly), img_shift(cb, 1, Ly)));
            if (DIM == 3) dz = sub2(dz, pk(img_shift(ca, 2, Lz), img_shift(cb, 2, Lz)));
        }
        const float2 r2 = fma2(dz, dz, fma2(dy, dy, mul2(dx, dx)));
        ha = ha && r2.x < (VARH ? pair_cut2(kh, hi, a.pj.w) : cut2c);
        hb = hb && r2.y < (VARH ? pair_cut2(kh, hi, b.pj.w) : cut2c);
        if (FILTER) { ha = ha && ((my_mask >> a.aid) & 1u); hb = hb && ((my_mask >> b.aid) & 1u); }
        nhits += (ha ? 1u : 0u) + (hb ? 1u : 0u);
        const float2 rinv = pk(r2.x > 0.0f ? rsqrt_approx(r2.x) : 0.0f, r2.y > 0.0f ? rsqrt_approx(r2.y) : 0.0f);
        const float2 r = mul2(r2, rinv);
        float2 hinv, mfac;
        if (VARH) {
            hinv = rcp2(mul2(pk1(0.5f), add2(pk1(hi), pk(a.pj.w, b.pj.w))));
            const float2 m2 = UM ? pk1(pc.m_const) : pk(a.mj, b.mj);
            mfac = mul2(mul2(m2, pk1(sigma)), DIM == 3 ? mul2(mul2(hinv, hinv), hinv) : mul2(hinv, hinv));
        } else { hinv = pk1(hinv_c); mfac = UM ? pk1(mfac_c) : mul2(pk(a.pj.w, b.pj.w), pk1(fac_c)); }
        float2 f, df;
        kernel_profile2<KERNEL, DIM>(mul2(r, hinv), f, df);
        mfac = pk(ha ? mfac.x : 0.0f, hb ? mfac.y : 0.0f);              // a candidate that fails contributes nothing
        rho2 = fma2(mfac, f, rho2);
#ifdef SPH_EXP_RED
        // EXPERIMENT (DESIGN.md "Tried and dropped" (g)): the cost of ONE red.global.add.f32 per true pair, which a
        // symmetric once-per-pair density pass would need for the j side (the target word is scratch: acc.w)
        if (ha) atomicAdd(&S.acc[a.j].w, mfac.x * f.x);
        if (hb) atomicAdd(&S.acc[b.j].w, mfac.y * f.y);
#endif
    };
#endif

    TileState st; st.reset(); st.tests = 0;
    const uint32_t idle = in ? (uint32_t)i : 0u;
    auto drain = [&](uint32_t nz, bool shifted) {
#ifdef SPH_REAL_DOUBLE
        if (shifted) tile_drain<DensitySrc, 2, true>(ws, nz, idle, load, compute);
        else         tile_drain<DensitySrc, 2, false>(ws, nz, idle, load, compute);
#else
        if (shifted) tile_drain2<DensitySrc, TILE_DRAIN_DEPTH_DENSITY, true>(ws, nz, idle, load, compute);
        else         tile_drain2<DensitySrc, TILE_DRAIN_DEPTH_DENSITY, false>(ws, nz, idle, load, compute);
#endif
    };
    const uint32_t head = REPLAY ? __ldg(nl.head + warp_id) : SPH_NL_NONE;
    if (head != SPH_NL_NONE) {
        tile_replay(g, nl, head, ws, active, drain);
    } else {                                    // no record (or one that did not fit the pool): search
        tile_walk<DIM, VARH>(g, pc, S.posh, cell_start, active, in, to_float4(pi), ci, ws, st, [&]() { drain(st.nz, st.shifted); st.reset(); });
    }

    if (active) {
#ifndef SPH_REAL_DOUBLE
        const real rho = rho2.x + rho2.y;
#endif
        const real p = eos_pressure(rho, pc.rho0, pc.B, pc.gamma, pc.gamma_is_7);
        S.rp[i] = make_real2(rho, p / (rho * rho));
        if (!VARH || UM) S.velm[i].w = rho;                             // constant h, or VU layout: velm.w carries rho (SortedState)
        if (UM && !VARH) S.posh[i].w = p / (rho * rho);                 // UM layout: posh.w carries p/rho^2
        if (!isfinite(rho) || !(rho > real(0))) atomicAdd(&counters[CNT_NONFINITE], 1ull);
    }
    const unsigned long long h = warp_sum_u64(nhits), t = warp_sum_u64((unsigned long long)st.tests);
    if ((threadIdx.x & 31) == 0) { atomicAdd(&counters[CNT_PAIRS_DENSITY], h); atomicAdd(&counters[CNT_CAND_DENSITY], t); }
}

template <int KERNEL, int DIM>
static int launch_density_tile_kd(sph_ctx* c, bool filter, bool replay) {
    const int n = (int)c->n_total;
    if (n == 0) return SPH_OK;
    const int grid = (n + TILE_BLOCK - 1) / TILE_BLOCK;
    SortedState& S = c->S[c->cur];
#define LD(VARH, FILTER, REPLAY, UM) \
        SPH_LAUNCH(c, (REPLAY ? SPH_K_DENSITY_LIST : SPH_K_DENSITY), (k_density_tile<KERNEL, DIM, VARH, FILTER, REPLAY, UM>), grid, TILE_BLOCK, 0, c->grid, c->pc, S, c->cell_start, n, c->nl, c->counters)
#define LD2(VARH, FILTER, UM) do { if (replay) LD(VARH, FILTER, true, UM); else LD(VARH, FILTER, false, UM); } while (0)
#define LD3(VARH, UM) do { if (filter) LD2(VARH, true, UM); else LD2(VARH, false, UM); } while (0)
    if (c->variable_h) { if (c->pc.varh_um) LD3(true, true); else LD3(true, false); } else if (c->pc.uniform_m) LD3(false, true); else LD3(false, false);
#undef LD3
#undef LD2
#undef LD
    return SPH_OK;
}

// One launch computes rho,p for every array whose src_mask_per_dest entry is non-zero; it replays the records of
// launch_search when they match the current sorted order and searches itself otherwise.
int launch_density(sph_ctx* c, const uint32_t* src_mask_per_dest) {
    bool filter = false;
    for (int a = 0; a < SPH_MAX_ARRAYS; ++a) {
        c->pc.src_mask[a] = a < c->na ? src_mask_per_dest[a] : 0u;
        if (c->pc.src_mask[a] && c->pc.src_mask[a] != c->pc.all_mask) filter = true;
    }
    const bool replay = c->nl_valid && c->nl.pool != nullptr;
    const int k = c->prm.kernel, d = c->grid.dim;
    int rc = sph_fail(c, SPH_ERR_BAD_ARG, "unsupported kernel/dim");
#define KD(K, D) if (k == K && d == D) rc = launch_density_tile_kd<K, D>(c, filter, replay)
    KD(SPH_KERNEL_CUBIC, 2); KD(SPH_KERNEL_CUBIC, 3);
    KD(SPH_KERNEL_QUINTIC, 2); KD(SPH_KERNEL_QUINTIC, 3);
    KD(SPH_KERNEL_WENDLAND_C2, 2); KD(SPH_KERNEL_WENDLAND_C2, 3);
#undef KD
    return rc;
}
