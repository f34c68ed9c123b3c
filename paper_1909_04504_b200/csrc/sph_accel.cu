// WCSPH acceleration, eq.8-9 (L128-132; Listing 4):
//     a_i = g - sum_j m_j (p_i/rho_i^2 + p_j/rho_j^2 + Pi_ij) grad_i W_ij
// with Monaghan artificial viscosity Pi_ij (R9; the paper only names "the classic scheme", L185)
// and, in the same pair loop ("no inter-dependencies and may be computed together", L337), the continuity
// right-hand side eq.7 (L126; Listing 4):   arho_i = sum_j m_j (v_i - v_j) . grad_i W_ij.
// Gravity is the initial value of the accumulator (Listing 4).  With sph_params.nu > 0 the laminar
// viscosity of eq.10 (L134-136) is added in the same loop (LAMINAR instantiations).
#include "sph_tile.cuh"

// One kernel, two modes (sph_tile.cuh).  REPLAY = false: the warp searches its own candidates (no record pool).
// REPLAY = true: it replays the candidate masks recorded by launch_search for this sorted order and walks
// nothing (a warp whose record did not fit the pool searches).  Destination arrays named in
// arho_only_arrays serve ContinuityEquation(dest=solid, sources=[fluid]) (Listing 3): the same loop,
// only arho is stored; they share the launch with the momentum destinations.
// This file is compiled four times (build.py): once per smoothing kernel with -DSPH_ACCEL_KERNEL=<id> (the kernel
// template and its launcher launch_accel_k<id>), and once without (the dispatcher launch_accel).
int launch_accel_k0(sph_ctx* c, int dim, bool filter, bool want_arho, const AccelRoles& roles, bool replay);
int launch_accel_k1(sph_ctx* c, int dim, bool filter, bool want_arho, const AccelRoles& roles, bool replay);
int launch_accel_k2(sph_ctx* c, int dim, bool filter, bool want_arho, const AccelRoles& roles, bool replay);

#ifdef SPH_ACCEL_KERNEL
struct AccelSrc { real4 pj, vj; real2 rj; uint32_t aid; };

template <int KERNEL, int DIM, bool VARH, bool ARHO, bool FILTER, bool REPLAY, int PM, bool LAMINAR>
__global__ void __launch_bounds__(TILE_BLOCK, TILE_MIN_BLOCKS_ACCEL)
k_accel_tile(GridDesc g, PairConsts pc, SortedState S, const uint32_t* __restrict__ cell_start, int n,
             AccelRoles roles, NList nl, unsigned long long* __restrict__ counters) {
    typedef TileWarpSmemT<TILE_MMAX_OF(VARH)> WS;
    __shared__ WS smem[TILE_WARPS];
    WS& ws = smem[threadIdx.x >> 5];
    const int i = blockIdx.x * TILE_BLOCK + threadIdx.x;
    const int warp_id = i >> 5;
    const bool in = i < n;
    uint32_t meta = 0, ci = 0; real4 pi = make_real4(0, 0, 0, 1), vi = make_real4(0, 0, 0, 0);
    real2 ri = make_real2(1, 0);
    if (in) { meta = S.meta[i]; pi = ldg_r(S.posh + i); vi = ldg_r(S.velm + i); ri = ldg_r(S.rp + i); ci = S.cell[i]; }
    const uint32_t aid_i = meta >> SPH_META_IDX_BITS;
    const uint32_t my_mask = in ? pc.src_mask[aid_i] : 0u;
    const bool active = my_mask != 0u;
    // arrays that are no destination of any launch of this evaluation: their accelerations are zero (the sort does
    // not carry acc along, so what lies in their rows belongs to other particles)
    if (in && !active && (((roles.zero_xyz | roles.zero_w) >> aid_i) & 1u)) {
        real4 a = S.acc[i];
        if ((roles.zero_xyz >> aid_i) & 1u) { a.x = 0.0f; a.y = 0.0f; a.z = 0.0f; }
        if ((roles.zero_w >> aid_i) & 1u) a.w = 0.0f;
        S.acc[i] = a;
    }
    if (!__any_sync(SPH_FULL_MASK, active)) return;

    const real Lx = g.Lr[0], Ly = g.Lr[1], Lz = g.Lr[2];
    const real sigma = pc.sigma, h_c = pc.h_const, hinv_c = pc.hinv_const, fac_c = pc.fac_const;
    const real kh = sizeof(real) == 8 ? pc.ksup : pc.kh;               // what pair_cut2 of the build's real type takes
    const real visc = pc.visc, eps = pc.eps, nu4 = pc.nu4, eta = pc.eta;
    const real hi = VARH ? pi.w : h_c;
    const real cut2c = pair_cut2(kh, h_c, h_c);
    // Wendland-C2: sigma h^-(d+2) f'(q)/q = cw (1 - q/2)^3, times the mass where every particle has the same one
    constexpr bool MCONST = PM == 2 || (VARH && PM == 1);
    const real mw = MCONST ? pc.m_const : real(1);
    const real sigma5 = real(-5) * sigma * mw, cw_c = real(-5) * fac_c * hinv_c * hinv_c * mw;
    // PM: where the neighbour's rho and p/rho^2 come from (the loop is L1-gather bound: fewer gathers pay).
    //   0  gathered from rp (caller-supplied p, gamma != 7 ...): three gathers
    //   1  gamma = 7, every p is the EOS of its rho, and velm.w carries rho (constant h, or variable h with uniform
    //      mass): p/rho^2 is recomputed (the destination's own term too, so that the pair terms stay antisymmetric):
    //      two gathers
    //   2  UM layout (constant h, uniform mass): rho in velm.w, p/rho^2 in posh.w, m = m_const: two gathers
    const real inv_rho0 = 1.0f / pc.rho0, rho0 = pc.rho0, Beos = pc.B;
    const real rho_i = ri.x, pr_i = PM == 1 ? eos7_p_over_rho2(ri.x, rho0, inv_rho0, Beos) : ri.y;
    const real m_const = pc.m_const;
    real ax = pc.g[0], ay = pc.g[1], az = pc.g[2], ar = 0.0f;      // gravity = accumulator init (Listing 4)
    unsigned nhits = 0;                                                 // pairs that pass the exact predicate (and the source mask)
    auto load = [&](uint32_t j) {
        SPH_DBG_ASSERT(j < g.n_sorted, g);
        AccelSrc s; s.pj = ldg_r(S.posh + j); s.vj = ldg_r(S.velm + j); s.aid = 0u;
        s.rj = PM ? make_real2(0.0f, 0.0f) : ldg_r(S.rp + j);
        if (FILTER) { if (my_mask != pc.all_mask) s.aid = __ldg(S.meta + j) >> SPH_META_IDX_BITS; }   // lanes fed by all arrays skip the gather
        return s;
    };
    auto compute = [&](const AccelSrc& s, bool has, uint32_t code, auto per) {
        // the exact predicate of DESIGN.md R7 on the candidate the tensor-core filter let through
        real dx = rsub(pi.x, s.pj.x), dy = rsub(pi.y, s.pj.y), dz = DIM == 3 ? rsub(pi.z, s.pj.z) : real(0);
        if (decltype(per)::value) {
            dx = rsub(dx, img_shift(code, 0, Lx)); dy = rsub(dy, img_shift(code, 1, Ly));
            if (DIM == 3) dz = rsub(dz, img_shift(code, 2, Lz));
        }
        const real r2 = pair_r2(dx, dy, dz);
        has = has && r2 < (VARH ? pair_cut2(kh, hi, s.pj.w) : cut2c);
        if (FILTER) has = has && (my_mask == pc.all_mask || ((my_mask >> s.aid) & 1u));
        nhits += has ? 1u : 0u;
        real hij, hinv;
        if (VARH) { hij = 0.5f * (hi + s.pj.w); hinv = rcp_approx(hij); } else { hij = h_c; hinv = hinv_c; }
        // SortedState layouts: where m, rho and p/rho^2 of the neighbour ride
        const real mj = PM == 2 ? m_const : (VARH ? (PM == 1 ? m_const : s.vj.w) : s.pj.w);
        real mgc;                                                       // m_j grad_i W_ij = mgc * (dx,dy,dz)
        if (KERNEL == SPH_KERNEL_WENDLAND_C2 && DIM > 1) {
            // f'(q)/q = -5 (1 - q/2)^3 is a polynomial, so sigma h^-(d+2) f'(q)/q needs no 1/r (at r = 0 the term
            // vanishes with dx = dy = dz = 0, R18); a uniform mass rides in the constant
            const real t = rmax(rfma(real(-0.5), sqrt_approx(r2) * hinv, real(1)), real(0));
            const real hinv2 = hinv * hinv;
            const real cw = VARH ? sigma5 * (hinv2 * hinv2) * (DIM == 3 ? hinv : real(1)) : cw_c;
            mgc = cw * (t * t * t);
            if (!MCONST) mgc *= mj;
        } else {
            const real rinv = r2 > 0.0f ? rsqrt_approx(r2) : real(0);   // grad W := 0 at r = 0 (R18): rinv = 0
            const real fac = VARH ? sigma * hinv * hinv * (DIM == 3 ? hinv : real(1)) : fac_c;
            real f, df;
            kernel_profile<KERNEL, DIM>(r2 * rinv * hinv, f, df);
            mgc = mj * (fac * hinv * df * rinv);
        }
        const real vx = vi.x - s.vj.x, vy = vi.y - s.vj.y;
        real vr = rfma(vy, dy, vx * dx);
        if (DIM == 3) vr = rfma(vi.z - s.vj.z, dz, vr);
        const real rho_j = PM ? s.vj.w : s.rj.x;
        const real pr_j = PM == 2 ? s.pj.w : (PM == 1 ? eos7_p_over_rho2(rho_j, rho0, inv_rho0, Beos) : s.rj.y);
        // Pi_ij = -alpha c0 mu / rhobar, mu = h vr/(r^2 + eps h^2), rhobar = (rho_i+rho_j)/2, only if vr < 0
        const real den = rfma(eps * hij, hij, r2) * (rho_i + rho_j);
        const real Pi = vr < real(0) ? visc * hij * vr * rcp_approx(den) : real(0);
        const real mg = has ? mgc : real(0);                              // a lane that has run out contributes nothing
        const real sc = -mg * (pr_i + pr_j + Pi);
        ax = rfma(sc, dx, ax); ay = rfma(sc, dy, ay);
        if (DIM == 3) az = rfma(sc, dz, az);
        if (ARHO) ar = rfma(mg, vr, ar);
        if (LAMINAR) {                                                  // laminar viscosity, eq.10 (launches with nu != 0)
            // m_j 4nu/(rho_i+rho_j) (r.gradW)/(r^2 + eta h^2) u_ij,  r.gradW = gc r^2
            const real lam = mg * nu4 * r2 * rcp_approx(rmax(rfma(eta * hij, hij, r2) * (rho_i + rho_j), real(1.0e-30)));
            ax = rfma(lam, vx, ax); ay = rfma(lam, vy, ay);
            if (DIM == 3) az = rfma(lam, vi.z - s.vj.z, az);
        }
    };
    const uint32_t idle = in ? (uint32_t)i : 0u;
    constexpr int DEPTH = REPLAY ? TILE_DRAIN_DEPTH_REPLAY : 2;
    auto drain = [&](uint32_t nz, bool shifted) {
        if (shifted) tile_drain<AccelSrc, DEPTH, true>(ws, nz, idle, load, compute);
        else         tile_drain<AccelSrc, DEPTH, false>(ws, nz, idle, load, compute);
    };

    TileState st; st.reset(); st.tests = 0;
    const uint32_t head = REPLAY ? __ldg(nl.head + warp_id) : SPH_NL_NONE;
    if (head != SPH_NL_NONE) {
        tile_replay(g, nl, head, ws, active, drain);
    } else {                                    // no record (or one that did not fit the pool): search
        tile_walk<DIM, VARH>(g, pc, S.posh, cell_start, active, in, to_float4(pi), ci, ws, st, [&]() { drain(st.nz, st.shifted); st.reset(); });
    }
    if (active) {
        real4 a;
        if ((roles.arho_only >> aid_i) & 1u) {                          // ContinuityEquation-only destination array
            a = ((roles.keep_xyz >> aid_i) & 1u) ? S.acc[i] : make_real4(0.0f, 0.0f, 0.0f, 0.0f);
            a.w = ar;
        } else a = make_real4(ax, ay, DIM == 3 ? az : real(0), ARHO ? ar : real(0));
        S.acc[i] = a;
        if (!isfinite(a.x) || !isfinite(a.y) || !isfinite(a.z) || !isfinite(a.w)) atomicAdd(&counters[CNT_NONFINITE], 1ull);
    }
    const unsigned long long h = warp_sum_u64(nhits), t = warp_sum_u64((unsigned long long)st.tests);
    if ((threadIdx.x & 31) == 0) { atomicAdd(&counters[CNT_PAIRS_ACCEL], h); if (t) atomicAdd(&counters[CNT_CAND_ACCEL], t); }
}

template <int KERNEL, int DIM>
static int launch_accel_tile_kd(sph_ctx* c, bool filter, bool want_arho, const AccelRoles& roles, bool replay) {
    const int n = (int)c->n_total;
    if (n == 0) return SPH_OK;
    const bool varh = c->variable_h;
    SortedState& S = c->S[c->cur];
    const int grid = (n + TILE_BLOCK - 1) / TILE_BLOCK;
    // velm.w carries rho when h is constant or every mass is equal (SortedState)
    const bool eos7 = c->p_is_eos && c->pc.gamma_is_7;
    const int pm = varh ? (c->pc.varh_um ? 1 : 0) : (c->pc.uniform_m ? 2 : (eos7 ? 1 : 0));
    const bool lam = c->pc.nu4 != 0.0f;
#define LT(VARH, ARHO, FILTER, REPLAY, PM, LAM) \
        SPH_LAUNCH(c, (REPLAY ? SPH_K_ACCEL_LIST : SPH_K_ACCEL), (k_accel_tile<KERNEL, DIM, VARH, ARHO, FILTER, REPLAY, PM, LAM>), grid, TILE_BLOCK, 0, c->grid, c->pc, S, c->cell_start, n, roles, c->nl, c->counters)
#define LT0(VARH, ARHO, FILTER, REPLAY, PM) do { if (lam) LT(VARH, ARHO, FILTER, REPLAY, PM, true); else LT(VARH, ARHO, FILTER, REPLAY, PM, false); } while (0)
#define LT1(VARH, ARHO, FILTER, PM) do { if (replay) LT0(VARH, ARHO, FILTER, true, PM); else LT0(VARH, ARHO, FILTER, false, PM); } while (0)
#define LT2(VARH, ARHO, PM) do { if (filter) LT1(VARH, ARHO, true, PM); else LT1(VARH, ARHO, false, PM); } while (0)
#define LT3(VARH, PM) do { if (want_arho) LT2(VARH, true, PM); else LT2(VARH, false, PM); } while (0)
    if (varh) { if (pm == 1) LT3(true, 1); else LT3(true, 0); } else if (pm == 2) LT3(false, 2); else if (pm == 1) LT3(false, 1); else LT3(false, 0);
#undef LT3
#undef LT2
#undef LT1
#undef LT0
#undef LT
    return SPH_OK;
}

#define SPH_CAT2(a, b) a##b
#define SPH_CAT(a, b) SPH_CAT2(a, b)
int SPH_CAT(launch_accel_k, SPH_ACCEL_KERNEL)(sph_ctx* c, int dim, bool filter, bool want_arho, const AccelRoles& roles, bool replay) {
    return dim == 2 ? launch_accel_tile_kd<SPH_ACCEL_KERNEL, 2>(c, filter, want_arho, roles, replay)
                    : launch_accel_tile_kd<SPH_ACCEL_KERNEL, 3>(c, filter, want_arho, roles, replay);
}

#else
// One launch serves every destination array whose mask is non-zero.  roles.arho_only: bit a = array a stores only
// its continuity sum (ContinuityEquation(dest=solid, sources=[fluid]), Listing 3).
int launch_accel(sph_ctx* c, const uint32_t* src_mask_per_dest, bool want_arho, const AccelRoles& roles) {
    bool filter = false;
    const bool use_list = c->nl_valid && c->nl.pool != nullptr;     // records of launch_search for this sorted order
    for (int a = 0; a < SPH_MAX_ARRAYS; ++a) {
        c->pc.src_mask[a] = a < c->na ? src_mask_per_dest[a] : 0u;
        if (c->pc.src_mask[a] && c->pc.src_mask[a] != c->pc.all_mask) filter = true;
    }
    c->last_used_rows = use_list;
    const int k = c->prm.kernel, d = c->grid.dim;
    if (d != 2 && d != 3) return sph_fail(c, SPH_ERR_BAD_ARG, "unsupported kernel/dim");
    const bool wa = want_arho || roles.arho_only != 0u;
    if (k == SPH_KERNEL_CUBIC)       return launch_accel_k0(c, d, filter, wa, roles, use_list);
    if (k == SPH_KERNEL_QUINTIC)     return launch_accel_k1(c, d, filter, wa, roles, use_list);
    if (k == SPH_KERNEL_WENDLAND_C2) return launch_accel_k2(c, d, filter, wa, roles, use_list);
    return sph_fail(c, SPH_ERR_BAD_ARG, "unsupported kernel/dim");
}
#endif
