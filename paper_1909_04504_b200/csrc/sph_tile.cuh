// Warp-tile pair machinery: candidate walk, tensor-core filter, hit masks, drain,
// mask records.
//
// Mapping.  A warp owns 32 consecutive particles of the CELL-SORTED order (level-major, x sub-cell fastest), i.e.
// a short tube along x inside one stencil row of its level grid (Fig.1).  Lanes of one level and
// row without a wide x gap form a GROUP.  For every group and every level b of the grid (one level when h is
// constant; PAPER.md L158-160, L171 for variable h) the candidates are the cells of level b that meet the
// group's bounding box grown by the reach R = k (h_group_max + h_max,b) / 2: a (rows in y) x (rows in z) set of
// stencil rows, each ONE contiguous run of the sorted order (+ the images across a periodic seam as separate runs
// with their shift code).  32 lanes look the runs up in parallel, one flat loop streams them 32 candidates at a
// time; the next batch is prefetched into registers while the current one is tested.
//
// Phase 1 (filter).  The 32 x 32 squared distances of a batch are a small dense contraction,
//     s_ij = |x_i - x_j|^2 - cut_ij^2 = n_i + n_j - 2 x_i . x_j - 2 kh^2 h_i h_j ,   n = |x|^2 - kh^2 h^2 ,
// so it runs on the tensor cores: 8 mma.sync.m16n8k8 (tf32 operands, fp32 accumulators) per batch, operands
// [-2x, -2y, -2z, -2 kh^2 h, n_hi, n_lo, 1, 1] . [x, y, z, h, 1, 1, n_hi, n_lo] in coordinates relative to the
// group's centre, rounded to tf32 (n split into two tf32 words).  tf32 cannot decide the bit-specified predicate
// of DESIGN.md R7, so the tensor-core result is only a CONSERVATIVE filter: a margin that bounds the rounding
// (derived in DESIGN.md "Tensor-core filter") is subtracted on the candidate side, the sign bits of the
// accumulators are collected with one funnel shift each, and a 4 x 4 byte transpose inside every quad gives each
// lane the 32-bit mask of ITS particle for the batch: a superset of its neighbours (+ 2-4 %).
// Phase 2 (evaluation).  When the mask store is full, and once at the end, the warp drains it: every lane pops its
// own candidates in order, applies the EXACT float predicate R7 (image-specific shift, fl(x_i - x_j), fma chain,
// r2 < cut2) and runs the expensive body (kernel, EOS terms, viscosity) on the true neighbours, so the body runs at
// mean/max neighbour-count lane utilisation instead of the hit rate of the tests.  Set membership is therefore
// decided by exactly the expression the oracle uses; the filter only has to have no false negatives.
// Records.  The search kernel (sph_search.cu) copies the masks, bases and shift codes (not the hit indices: 4 B per
// 32 tests instead of 4 B per hit) to the record pool, once per sorted order; the density and momentum passes
// replay them (tile_replay: one bulk copy per block), apply the exact predicate and walk nothing.
#pragma once
#include "sph_ctx.cuh"
#include <cstddef>
#include <type_traits>

#define TILE_BLOCK 128
#define TILE_WARPS (TILE_BLOCK / 32)
#ifndef TILE_MIN_BLOCKS
#define TILE_MIN_BLOCKS 8                 // resident blocks per SM the pair kernels are compiled for (64 registers)
#endif
#ifndef TILE_MIN_BLOCKS_DENSITY
#define TILE_MIN_BLOCKS_DENSITY 8
#endif
#ifndef TILE_MIN_BLOCKS_ACCEL
#define TILE_MIN_BLOCKS_ACCEL 6           // the momentum kernel is faster with 80 registers and 6 blocks (measured, C3, C4)
#endif
#ifndef TILE_DRAIN_DEPTH_REPLAY
#define TILE_DRAIN_DEPTH_REPLAY 3         // candidates in flight in the replaying momentum kernel
#endif
#ifndef TILE_DRAIN_DEPTH_DENSITY
#define TILE_DRAIN_DEPTH_DENSITY 2        // PAIRS of candidates in flight in the density drain
#endif
// masks per warp before a forced drain / per record block (<= 30: 30 bases + 2 words = one header row).  Constant h:
// 24 (a C3 / C4 tile streams ~22 batches; 30 costs a shared-memory carve-out step: C4 momentum 1.21 -> 1.36 ms);
// variable h: 30 (a C5 tile streams ~33: C5 13.6 -> 13.0 ms/step)
#ifndef TILE_MMAX_CONSTH
#define TILE_MMAX_CONSTH 24
#endif
#ifndef TILE_MMAX_VARH
#define TILE_MMAX_VARH 30
#endif
#define TILE_MMAX_OF(VARH) ((VARH) ? TILE_MMAX_VARH : TILE_MMAX_CONSTH)

template <int MM>
struct __align__(16) TileWarpSmemT {
    static constexpr int MMAX = MM;
    // the image of one record block, in the layout of the pool (so that a replaying warp fetches a block with ONE
    // bulk copy): header row, shift-code row, mask rows
    uint32_t hdr[32];                      // [0] next block, [1] batches | flags, [2 + m] first sorted index of batch m
    uint32_t bcode[32];                    // image-shift code of every batch (2 bits per axis: 1 -> -L, 2 -> +L)
    uint32_t mask[MM][32];                 // candidate masks, [batch][lane]: bit 31 - c = candidate c of the batch (most
                                           // significant bit first, so that a pop is one count-leading-zeros)
    // Directly behind the masks, so that zero_row is "mask row MM": the row the sentinel bit of nz points at.  The
    // drains clear it when they start; G / Af are dead while a drain runs (every batch stages G anew).
    union {
        float2 G[4][34];                   // B operands of one batch: G[t][c] = (feature t, feature t+4) of the candidate in column c
        float Af[32 * 9];                  // A operands of a group while the quads exchange them (stride 9: conflict-free)
        uint32_t zero_row[32];
    };
    unsigned long long bar;                // mbarrier of the bulk copy
    uint32_t seg_s[32], seg_e[32], seg_c[32];   // candidate runs of the current pass: [s, e) and image-shift code
    // warp-uniform walker state that only the (cold) group / level / pass set-up code touches: kept here, not in
    // registers, so that the batch loop stays within the register budget
    float bb[8];                           // group bounding box xmin, xmax, ymin, ymax, zmin, zmax, largest h, half extent
    int lv[8];                             // level ranges x0, x1, y0, z0, ny, entries, nparts | low << 8 | high << 9
    float inv_ny;
    // mask row m of this lane, m in [0, MM]; row MM is the zero row
    __device__ __forceinline__ uint32_t mask_row(int m, int lane) const { return (&mask[0][0])[m * 32 + lane]; }
};

static_assert(offsetof(TileWarpSmemT<TILE_MMAX_VARH>, zero_row) == offsetof(TileWarpSmemT<TILE_MMAX_VARH>, mask) + TILE_MMAX_VARH * 128 &&
              offsetof(TileWarpSmemT<TILE_MMAX_CONSTH>, zero_row) == offsetof(TileWarpSmemT<TILE_MMAX_CONSTH>, mask) + TILE_MMAX_CONSTH * 128 &&
              offsetof(TileWarpSmemT<TILE_MMAX_VARH>, hdr) == 0 && TILE_MMAX_VARH <= 30 && TILE_MMAX_CONSTH <= 30,
              "record block image at offset 0; the zero row directly behind the mask rows");

struct TileState {
    int M;                                 // masks stored since the last drain (warp-uniform)
    uint32_t nz;                           // bit 31 - m: this lane's mask m is not empty
    bool shifted;                          // some stored batch came from a periodic image (warp-uniform)
    unsigned tests;                        // candidates streamed for this lane's particle
    __device__ __forceinline__ void reset() { M = 0; nz = 0u; shifted = false; }
};

// plain (coherent) loads of the sorted state: the density pass rewrites .w words of records that other warps gather
template <class T> __device__ __forceinline__ T ld_state(const T* p) { return *p; }

__device__ __forceinline__ float tf32r(float x) {           // round to tf32 (10 explicit mantissa bits), half away from zero
    return __uint_as_float((__float_as_uint(x) + 0x1000u) & 0xffffe000u);
}
__device__ __forceinline__ uint32_t f2ord(float x) {         // order-preserving float -> uint
    const uint32_t b = __float_as_uint(x);
    return b ^ ((uint32_t)((int32_t)b >> 31) | 0x80000000u);
}
__device__ __forceinline__ float ord2f(uint32_t o) {
    return __uint_as_float(o ^ (((o >> 31) - 1u) | 0x80000000u));
}
__device__ __forceinline__ float warp_min_f(float v) { return ord2f(__reduce_min_sync(SPH_FULL_MASK, f2ord(v))); }
__device__ __forceinline__ float warp_max_f(float v) { return ord2f(__reduce_max_sync(SPH_FULL_MASK, f2ord(v))); }

// x >> s with the hardware's semantics for s >= 32 (0), which C++ leaves undefined
__device__ __forceinline__ uint32_t shr_u32(uint32_t x, int s) {
    uint32_t r; asm("shr.u32 %0, %1, %2;" : "=r"(r) : "r"(x), "r"(s)); return r;
}

// minimum-image shift of a batch on one axis from its code: d = fl(x_i - x_j) - shift (R7)
template <class T>
__device__ __forceinline__ T img_shift(uint32_t code, int axis, T L) {
    const T lo = (code & (1u << (2 * axis))) ? -L : T(0);           // two selects on single bits: no branch per candidate
    return (code & (2u << (2 * axis))) ? L : lo;
}

// D = A (16 x 8, tf32, row) * B (8 x 8, tf32, col), fp32 accumulators starting from zero
__device__ __forceinline__ void mma_tf32_16x8x8(float (&c)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
    asm("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%10,%10,%10,%10};"
        : "=f"(c[0]), "=f"(c[1]), "=f"(c[2]), "=f"(c[3])
        : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1), "f"(0.0f));
}

// Walks every candidate run of the warp's 32 particles.  `drain()` is called (warp-uniformly, from ONE site)
// whenever the mask store holds WS::MMAX batches, and once at the end; it must consume the masks and call
// st.reset().  All 32 lanes must call this.   in: the lane holds a particle; active: it is a destination of this
// launch; pi = (x, y, z, h); ci = its cell id (level base + linear cell).
template <int DIM, bool VARH, class WS, class Drain>
__device__ __forceinline__ void tile_walk(const GridDesc& g, const PairConsts& pc,
                                          const real4* posh, const uint32_t* __restrict__ cell_start,
                                          bool active, bool in, float4 pi, uint32_t ci,
                                          WS& ws, TileState& st, Drain&& drain) {
    const int lane = threadIdx.x & 31, gq = lane >> 2, tq = lane & 3;
    const int na = g.na, nlev = VARH ? g.nlev : 1;
    // the search runs in float whatever the real type of the build (see sph_internal.cuh)
    const float khf = (float)pc.kh, hcf = (float)pc.h_const;
    const float khsq = khf * khf;
    const float cut2c = pair_cut2(khf, hcf, hcf);

    // own cell -> (level, stencil row, x sub-cell); groups: maximal lane ranges of one level and row without an x
    // gap wider than two coarse cells (a wider gap means the windows of its two sides are disjoint)
    int lvl = 0;
    if (VARH) { while (lvl + 1 < nlev && ci >= g.lev[lvl + 1].base) ++lvl; }
    const uint32_t rel = ci - g.lev[lvl].base;
    const uint32_t nc0_own = (uint32_t)g.lev[lvl].nc[0];
    int row = in ? (int)(rel / nc0_own) : -1;
    const int sub = in ? (int)(rel % nc0_own) : 0;
    const int gap = 2 * g.lev[lvl].xsub;
    if (VARH) row = in ? row * SPH_MAX_LEVELS + lvl : -1;                 // rows of different levels never compare equal
    const int prow = __shfl_up_sync(SPH_FULL_MASK, row, 1), psub = __shfl_up_sync(SPH_FULL_MASK, sub, 1);
    const bool brk = lane == 0 || row != prow || sub - psub > gap;
    const unsigned brkmask = __ballot_sync(SPH_FULL_MASK, brk);
    unsigned remaining = __ballot_sync(SPH_FULL_MASK, active);

    // per-thread constants of the mask transpose (two butterfly rounds inside the quad) and of the B-operand fetch
    const uint32_t sel1 = (tq & 1) ? 0x3715u : 0x6240u, sel2 = (tq & 2) ? 0x3276u : 0x5410u;
    const int cidx = 8 * (gq >> 1) + 7 - (gq & 1);           // column g of N-tile nt holds staged candidate cidx - 2 nt

    // ---- group state (warp-uniform unless noted); the cold part lives in ws.bb / ws.lv
    bool grp = false, ing = false /* per lane */;
    float ox = 0, oy = 0, oz = 0;
    uint32_t A0[4] = {0, 0, 0, 0}, A1[4] = {0, 0, 0, 0};      // per lane: A operands (rows of the quad's four particles)
    // ---- level state
    int b = 0, pass = 0, npass = 0;
    float nsub = 0.0f;                                         // subtracted on the candidate side: filter margin (+ cut^2 when h is constant)
    // ---- run / batch state
    unsigned segs = 0u;
    bool have = false;
    uint32_t nb0 = 0u, ne = 0u, ncode = 0u;
    float4 pjn = make_float4(0, 0, 0, 0);

    auto load_batch = [&](uint32_t bb, uint32_t ee) -> float4 {
        const uint32_t j = bb + (uint32_t)lane;
        SPH_DBG_ASSERT(ee <= g.n_sorted && bb <= ee, g);
        return j < ee ? to_float4(ld_state(posh + j)) : make_float4(0.0f, 0.0f, 0.0f, 0.0f);
    };
    auto pop_run = [&]() -> bool {
        if (!segs) return false;
        const int k = __ffs(segs) - 1; segs &= segs - 1u;
        nb0 = ws.seg_s[k]; ne = ws.seg_e[k]; ncode = ws.seg_c[k];
        return true;
    };

    auto setup_group = [&]() {
        const int leader = __ffs(remaining) - 1;
        const int gs = 31 - __clz(brkmask & (0xffffffffu >> (31 - leader)));      // start of the leader's range
        const unsigned above = leader < 31 ? (brkmask & (0xffffffffu << (leader + 1))) : 0u;
        const int ge = above ? __ffs(above) - 1 : 32;                               // one past its end
        const unsigned range = (ge == 32 ? 0xffffffffu : ((1u << ge) - 1u)) & (0xffffffffu << gs);
        const unsigned gmask = remaining & range;
        remaining &= ~gmask;
        ing = (gmask >> lane) & 1u;
        const float big = 3.0e38f;
        const float xmin = warp_min_f(ing ? pi.x : big), xmax = warp_max_f(ing ? pi.x : -big);
        const float ymin = warp_min_f(ing ? pi.y : big), ymax = warp_max_f(ing ? pi.y : -big);
        float zmin = 0.0f, zmax = 0.0f, hg = hcf;
        if (DIM == 3) { zmin = warp_min_f(ing ? pi.z : big); zmax = warp_max_f(ing ? pi.z : -big); }
        if (VARH) hg = __uint_as_float(__reduce_max_sync(SPH_FULL_MASK, ing ? __float_as_uint(pi.w) : 0u));
        ox = 0.5f * (xmin + xmax); oy = 0.5f * (ymin + ymax); oz = DIM == 3 ? 0.5f * (zmin + zmax) : 0.0f;
        // A operands of this lane's particle: [-2x, -2y, -2z, -2 kh^2 h, n_hi, n_lo, 1, 1], n = |x|^2 - kh^2 h^2
        const float xt = tf32r(pi.x - ox), yt = tf32r(pi.y - oy), zt = DIM == 3 ? tf32r(pi.z - oz) : 0.0f;
        const float ht = VARH ? tf32r(pi.w) : 0.0f;
        const float n = fmaf(zt, zt, fmaf(yt, yt, xt * xt)) - khsq * ht * ht;
        const float nh = tf32r(n), nl = tf32r(n - nh);
        __syncwarp();                                          // G (aliased) is no longer read
        float* af = ws.Af + lane * 9;
        af[0] = -2.0f * xt; af[1] = -2.0f * yt; af[2] = -2.0f * zt; af[3] = tf32r(-2.0f * khsq * ht);
        af[4] = nh; af[5] = nl; af[6] = 1.0f; af[7] = 1.0f;
        if (lane == 0) {
            ws.bb[0] = xmin; ws.bb[1] = xmax; ws.bb[2] = ymin; ws.bb[3] = ymax; ws.bb[4] = zmin; ws.bb[5] = zmax; ws.bb[6] = hg;
            ws.bb[7] = 0.5f * fmaxf(fmaxf(xmax - xmin, ymax - ymin), DIM == 3 ? zmax - zmin : 0.0f);
        }
        __syncwarp();
        const float* q = ws.Af + (4 * gq) * 9 + tq;             // rows of the quad's particles 0..3, features tq and tq + 4
        A0[0] = __float_as_uint(q[0]);      A0[1] = __float_as_uint(q[9]);       A0[2] = __float_as_uint(q[4]);      A0[3] = __float_as_uint(q[13]);
        A1[0] = __float_as_uint(q[18]);     A1[1] = __float_as_uint(q[27]);      A1[2] = __float_as_uint(q[22]);     A1[3] = __float_as_uint(q[31]);
        __syncwarp();
    };

    // candidate cells of level b: the level's cells that meet the group's bounding box grown by the reach R
    auto setup_level = [&]() {
        const LevelDesc& Lv = g.lev[b];
        const float xmin = ws.bb[0], xmax = ws.bb[1], ymin = ws.bb[2], ymax = ws.bb[3], zmin = ws.bb[4], zmax = ws.bb[5];
        const float R = khf * (ws.bb[6] + (VARH ? Lv.hmax : hcf)) * 1.0001f + 16.0f * g.uabs;
        const float X = ws.bb[7] + R;                          // bound of every tile-local coordinate that matters
        // filter margin: bounds the tf32 rounding of operands and accumulation
        nsub = (R * X + R * R) * (1.0f / 256.0f) + X * X * (1.0f / 32768.0f) + 64.0f * g.uabs * (R + X) + (VARH ? 0.0f : cut2c);
        const int n0 = Lv.nc[0], n1 = Lv.nc[1], n2 = Lv.nc[2];
        const float e0 = 1.0e-3f + 4.8e-7f * (float)n0, e1 = 1.0e-3f + 4.8e-7f * (float)n1, e2 = 1.0e-3f + 4.8e-7f * (float)n2;
        int x0 = __float2int_rd((xmin - R - g.lo[0]) * Lv.inv_cell[0] - e0), x1 = __float2int_rd((xmax + R - g.lo[0]) * Lv.inv_cell[0] + e0);
        int y0 = __float2int_rd((ymin - R - g.lo[1]) * Lv.inv_cell[1] - e1), y1 = __float2int_rd((ymax + R - g.lo[1]) * Lv.inv_cell[1] + e1);
        int z0 = 0, z1 = 0;
        if (DIM == 3) { z0 = __float2int_rd((zmin - R - g.lo[2]) * Lv.inv_cell[2] - e2); z1 = __float2int_rd((zmax + R - g.lo[2]) * Lv.inv_cell[2] + e2); }
        if (!g.per[0]) { x0 = max(x0, 0); x1 = min(x1, n0 - 1); } else { x0 = max(x0, -n0); x1 = min(x1, 2 * n0 - 1); }
        if (!g.per[1]) { y0 = max(y0, 0); y1 = min(y1, n1 - 1); } else { y0 = max(y0, -n1); y1 = min(y1, 2 * n1 - 1); }
        if (DIM == 3) { if (!g.per[2]) { z0 = max(z0, 0); z1 = min(z1, n2 - 1); } else { z0 = max(z0, -n2); z1 = min(z1, 2 * n2 - 1); } }
        const bool lowpart = g.per[0] && x0 < 0, highpart = g.per[0] && x1 >= n0;
        const int nparts = 1 + (lowpart ? 1 : 0) + (highpart ? 1 : 0);
        const int ny = y1 - y0 + 1, nzr = z1 - z0 + 1;
        const int entries = (ny > 0 && nzr > 0 && x1 >= x0) ? ny * nzr * nparts : 0;
        npass = (entries + 31) >> 5;
        __syncwarp();
        if (lane == 0) {
            ws.lv[0] = x0; ws.lv[1] = x1; ws.lv[2] = y0; ws.lv[3] = z0; ws.lv[4] = ny; ws.lv[5] = entries;
            ws.lv[6] = nparts | (lowpart ? 0x100 : 0) | (highpart ? 0x200 : 0);
            ws.inv_ny = 1.0f / (float)max(ny, 1);
        }
        __syncwarp();
    };

    // 32 lanes look up 32 (row, x part) entries of the current level: [s, e) of the sorted order + shift code
    auto setup_pass = [&]() {
        const LevelDesc& Lv = g.lev[b];
        const int n0 = Lv.nc[0], n1 = Lv.nc[1], n2 = Lv.nc[2];
        const int x0 = ws.lv[0], x1 = ws.lv[1], y0 = ws.lv[2], z0 = ws.lv[3], ny = ws.lv[4], entries = ws.lv[5];
        const int nparts = ws.lv[6] & 0xff; const bool lowpart = (ws.lv[6] & 0x100) != 0;
        const int ent = pass * 32 + lane;
        bool nonempty = false;
        uint32_t s_ = 0u, e_ = 0u, code = 0u;
        if (ent < entries) {
            int r = ent, part = 0;
            if (nparts == 2) { r = ent >> 1; part = ent & 1; } else if (nparts == 3) { r = ent / 3; part = ent - 3 * r; }
            const int kind = part == 0 ? 0 : (part == 1 ? (lowpart ? 1 : 2) : 2);
            const int rz = (int)(((float)r + 0.5f) * ws.inv_ny);
            int iy = y0 + (r - rz * ny), iz = z0 + rz;
            if (iy < 0) { iy += n1; code |= 1u << 2; } else if (iy >= n1) { iy -= n1; code |= 2u << 2; }
            if (iz < 0) { iz += n2; code |= 1u << 4; } else if (iz >= n2) { iz -= n2; code |= 2u << 4; }
            int c0, c1;
            if (kind == 0)      { c0 = max(x0, 0); c1 = min(x1, n0 - 1); }
            else if (kind == 1) { c0 = max(x0 + n0, 0); c1 = n0 - 1; code |= 1u; }
            else                { c0 = 0; c1 = min(x1 - n0, n0 - 1); code |= 2u; }
            const uint32_t rowbase = Lv.base + (uint32_t)((iz * n1 + iy) * n0);
            SPH_DBG_ASSERT(c0 >= 0 && c0 <= c1 + 1 && c1 < n0 && iy >= 0 && iy < n1 && iz >= 0 && iz < n2 && rowbase + (uint32_t)c1 + 1u <= g.cells_total, g);
            s_ = __ldg(cell_start + (size_t)(rowbase + (uint32_t)c0) * na);
            e_ = __ldg(cell_start + (size_t)(rowbase + (uint32_t)c1 + 1u) * na);
            nonempty = s_ < e_;
        }
        __syncwarp();
        ws.seg_s[lane] = s_; ws.seg_e[lane] = e_; ws.seg_c[lane] = code;
        segs = __ballot_sync(SPH_FULL_MASK, nonempty);          // runs that hold candidates
        __syncwarp();
    };

    // one batch of <= 32 candidates [cb0, min(cb0 + 32, ce)) against the warp's 32 particles, in two parts so that the
    // prefetch of the next batch can overwrite the run state in place (no register copies of cb0 / ce / code / pj):
    // features(): this lane's candidate -> B-operand features + the batch's header words; filter(): staging, MMAs, masks
    struct Feat { float xt, yt, zt, ht, nh, nl; };
    auto features = [&](uint32_t cb0, uint32_t ce, uint32_t ccode, float4 pj) -> Feat {
        const bool valid = cb0 + (uint32_t)lane < ce;
        float xr = pj.x, yr = pj.y, zr = pj.z;
        if (ccode) {                                            // the image of the candidate next to the group: x_j + shift
            xr += img_shift(ccode, 0, g.L[0]); yr += img_shift(ccode, 1, g.L[1]);
            if (DIM == 3) zr += img_shift(ccode, 2, g.L[2]);
            st.shifted = true;
        }
        Feat f;
        f.xt = tf32r(xr - ox); f.yt = tf32r(yr - oy); f.zt = DIM == 3 ? tf32r(zr - oz) : 0.0f;
        f.ht = VARH ? tf32r(pj.w) : 0.0f;
        float n = fmaf(f.zt, f.zt, fmaf(f.yt, f.yt, f.xt * f.xt)) - (VARH ? khsq * f.ht * f.ht : 0.0f) - nsub;
        n = valid ? n : 1.0e30f;                                // padding never passes
        f.nh = tf32r(n); f.nl = tf32r(n - f.nh);
        if (lane == 0) { ws.hdr[2 + st.M] = cb0; ws.bcode[st.M] = ccode; }   // (slot M is free: the last drain consumed it)
        if (ing) st.tests += (unsigned)min(32u, ce - cb0);
        return f;
    };
    auto filter = [&](const Feat& f) {
        __syncwarp();                                           // readers of the previous batch are done
        const int slot = 31 - lane;                              // candidate c -> column 31 - c -> bit 31 - c of the masks
        ws.G[0][slot] = make_float2(f.xt, 1.0f); ws.G[1][slot] = make_float2(f.yt, 1.0f);
        ws.G[2][slot] = make_float2(f.zt, f.nh); ws.G[3][slot] = make_float2(f.ht, f.nl);
        __syncwarp();
        uint32_t pm0 = 0u, pm1 = 0u, pm2 = 0u, pm3 = 0u;        // sign bits of the quad's particles 0..3 (this thread's columns)
#pragma unroll
        for (int half = 0; half < 2; ++half) {                  // 4 independent MMAs in flight, then their 16 sign bits
            float c[2][2][4];
#pragma unroll
            for (int k = 0; k < 2; ++k) {
                const float2 bf = ws.G[tq][cidx - 2 * (2 * half + k)];
                mma_tf32_16x8x8(c[k][0], A0, __float_as_uint(bf.x), __float_as_uint(bf.y));
                mma_tf32_16x8x8(c[k][1], A1, __float_as_uint(bf.x), __float_as_uint(bf.y));
            }
#pragma unroll
            for (int k = 0; k < 2; ++k) {
                pm0 = __funnelshift_l(__float_as_uint(c[k][0][0]), pm0, 1); pm0 = __funnelshift_l(__float_as_uint(c[k][0][1]), pm0, 1);
                pm1 = __funnelshift_l(__float_as_uint(c[k][0][2]), pm1, 1); pm1 = __funnelshift_l(__float_as_uint(c[k][0][3]), pm1, 1);
                pm2 = __funnelshift_l(__float_as_uint(c[k][1][0]), pm2, 1); pm2 = __funnelshift_l(__float_as_uint(c[k][1][1]), pm2, 1);
                pm3 = __funnelshift_l(__float_as_uint(c[k][1][2]), pm3, 1); pm3 = __funnelshift_l(__float_as_uint(c[k][1][3]), pm3, 1);
            }
        }
        // byte q of P: this thread's 8 columns against particle q of the quad; transpose the 4 x 4 bytes of the quad
        // (byte k of lane t <- byte t of lane k) in two butterfly rounds: 2 x 2 bytes with lane ^ 1, halves with lane ^ 2
        const uint32_t P = __byte_perm(__byte_perm(pm0, pm1, 0x0040), __byte_perm(pm2, pm3, 0x0040), 0x5410);
        const uint32_t Rr = __byte_perm(P, __shfl_xor_sync(SPH_FULL_MASK, P, 1), sel1);
        uint32_t mask = __byte_perm(Rr, __shfl_xor_sync(SPH_FULL_MASK, Rr, 2), sel2);
        if (!ing) mask = 0u;
        ws.mask[st.M][lane] = mask;
        if (mask) st.nz |= 0x80000000u >> st.M;
        ++st.M;
    };

    // streams batches until the mask store is full (true) or every group is done (false)
    auto fill = [&]() -> bool {
        for (;;) {
            if (st.M >= WS::MMAX) return true;
            if (!have) {
                if (pop_run()) { pjn = load_batch(nb0, ne); have = true; continue; }
                if (grp) {
                    if (++pass < npass) { setup_pass(); continue; }
                    if (++b < nlev) { setup_level(); pass = -1; continue; }
                    grp = false;
                }
                if (!remaining) return false;
                setup_group(); grp = true; b = -1; npass = 0; pass = 0;
                continue;
            }
            const Feat f = features(nb0, ne, ncode, pjn);
            if (nb0 + 32u < ne) { nb0 += 32u; pjn = load_batch(nb0, ne); }     // prefetch the next batch
            else if (pop_run()) pjn = load_batch(nb0, ne);
            else have = false;
            filter(f);
        }
    };

    for (;;) {
        const bool more = fill();
        drain();                                                // consumes the masks, resets st
        if (!more) break;
    }
}

// Every lane pops its own candidates of the stored batches in order (nz: the lane's non-empty masks) and evaluates
// them.  A pop is two count-leading-zeros: masks and nz are stored most significant bit first, nz carries a
// sentinel bit that points at an all-zero mask row, so a lane that has run out needs no test of its own.  Branch-free and software-pipelined: DEPTH candidates are in flight, the source data of a later one is
// gathered (Src = load(sorted index)) before the current one is computed, so the gather latency overlaps the
// arithmetic.  A lane that has run out keeps executing with has = false and the harmless index `idle` (its own
// particle) until the slowest lane of the warp is done; compute(src, has, code, per) must apply the exact
// predicate and contribute nothing when it fails or has is false.  PER: some batch is a periodic image (code != 0).
template <class Src, int DEPTH, bool PER, class WS, class Load, class Compute>
__device__ __forceinline__ void tile_drain(WS& ws, uint32_t nz, uint32_t idle, Load&& load, Compute&& compute) {
    const int lane = threadIdx.x & 31;
    __syncwarp();
    uint32_t cur = 0u, b = 0u, code = 0u;
    constexpr uint32_t SENT = 0x80000000u >> WS::MMAX;      // sentinel: when the lane's masks are used up m = MMAX, the zero row
    ws.zero_row[lane] = 0u;                                 // (a lane reads its own column only: no warp sync needed)
    nz |= SENT;
    auto pop = [&](bool& has, uint32_t& cd) -> uint32_t {
        const bool refill = cur == 0u;
        const int m = __clz(nz);                            // the lane's next non-empty mask (bits are most significant first)
        const uint32_t nm = ws.mask_row(m, lane), nb = ws.hdr[2 + m];   // (m = MMAX: nb is a word of the next row, unused)
        cur = refill ? nm : cur; b = refill ? nb : b; nz = refill ? ((nz & shr_u32(0x7fffffffu, m)) | SENT) : nz;
        if (PER) { const uint32_t nc = ws.bcode[m]; code = refill ? nc : code; }
        has = cur != 0u;
        const int t = __clz(cur);                           // its next candidate; 32 when there is none
        const uint32_t j = has ? b + (uint32_t)t : idle;
        cur &= shr_u32(0x7fffffffu, t);                     // stays 0 when it is 0
        cd = code;
        return j;
    };
    Src R[DEPTH]; bool H[DEPTH]; uint32_t C[DEPTH];   // fully unrolled, so these live in registers
#pragma unroll
    for (int d = 0; d + 1 < DEPTH; ++d) R[d] = load(pop(H[d], C[d]));
    for (;;) {
#pragma unroll
        for (int d = 0; d < DEPTH; ++d) {
            const int nx = (d + DEPTH - 1) % DEPTH;
            R[nx] = load(pop(H[nx], C[nx]));        // gather for a later candidate ...
            compute(R[d], H[d], C[d], std::integral_constant<bool, PER>{});   // ... while this one is evaluated
        }
        if (!__any_sync(SPH_FULL_MASK, H[0])) break;   // pops are in order: no pending candidate 0 means none at all
    }
    __syncwarp();
}

// tile_drain2: as tile_drain, but every lane pops TWO candidates at a time and evaluates the pair with packed f32x2
// arithmetic (pays where the loop is bound by instruction issue: the density pass; the momentum pass is bound by
// its L1 gathers and stays scalar).  Branch-free and software-pipelined: DEPTH pairs are in
// flight, the source data of a later pair is gathered (Src = load(sorted index)) before the current one is
// computed, so the gather latency overlaps the arithmetic.  A lane that has run out keeps executing with has =
// false and the harmless index `idle` (its own particle) until the slowest lane of the warp is done;
// compute(srcA, srcB, hasA, hasB, codeA, codeB, per) must apply the exact predicate and contribute nothing where
// it fails or has is false.  PER: some batch is a periodic image (code != 0).
template <class Src, int DEPTH, bool PER, class WS, class Load, class Compute>
__device__ __forceinline__ void tile_drain2(WS& ws, uint32_t nz, uint32_t idle, Load&& load, Compute&& compute) {
    const int lane = threadIdx.x & 31;
    __syncwarp();
    uint32_t cur = 0u, b = 0u, code = 0u;
    constexpr uint32_t SENT = 0x80000000u >> WS::MMAX;      // sentinel: when the lane's masks are used up m = MMAX, the zero row
    ws.zero_row[lane] = 0u;                                 // (a lane reads its own column only: no warp sync needed)
    nz |= SENT;
    auto pop = [&](bool& has, uint32_t& cd) -> uint32_t {
        const bool refill = cur == 0u;
        const int m = __clz(nz);                            // the lane's next non-empty mask (bits are most significant first)
        const uint32_t nm = ws.mask_row(m, lane), nb = ws.hdr[2 + m];   // (m = MMAX: nb is a word of the next row, unused)
        cur = refill ? nm : cur; b = refill ? nb : b; nz = refill ? ((nz & shr_u32(0x7fffffffu, m)) | SENT) : nz;
        if (PER) { const uint32_t nc = ws.bcode[m]; code = refill ? nc : code; }
        has = cur != 0u;
        const int t = __clz(cur);                           // its next candidate; 32 when there is none
        const uint32_t j = has ? b + (uint32_t)t : idle;
        cur &= shr_u32(0x7fffffffu, t);                     // stays 0 when it is 0
        cd = code;
        return j;
    };
    Src R[DEPTH][2]; bool H[DEPTH][2]; uint32_t C[DEPTH][2];   // fully unrolled, so these live in registers
#pragma unroll
    for (int d = 0; d + 1 < DEPTH; ++d) { R[d][0] = load(pop(H[d][0], C[d][0])); R[d][1] = load(pop(H[d][1], C[d][1])); }
    for (;;) {
#pragma unroll
        for (int d = 0; d < DEPTH; ++d) {
            const int nx = (d + DEPTH - 1) % DEPTH;
            R[nx][0] = load(pop(H[nx][0], C[nx][0]));       // gathers for a later pair ...
            R[nx][1] = load(pop(H[nx][1], C[nx][1]));
            compute(R[d][0], R[d][1], H[d][0], H[d][1], C[d][0], C[d][1], std::integral_constant<bool, PER>{});   // ... while this one is evaluated
        }
        if (!__any_sync(SPH_FULL_MASK, H[0][0])) break;   // pops are in order: no pending candidate here means none at all
    }
    __syncwarp();
}

// ---- mask records (recorded by the search, replayed by the pair passes) ------------------------------------
// The pool is an array of ROWS of 32 words.  A warp appends BLOCKS of 2 + M rows: a header row {next block (row
// index, 0 = end), number of batches M <= WS::MMAX | 0x100 if a batch came from a periodic image, base[0..M-1]}, one
// row of shift codes (word = batch), then M rows of masks (word = lane).  A block is contiguous, so a replaying
// warp fetches it with ONE bulk copy (cp.async.bulk + mbarrier; SASS UBLKCP) into the same layout in shared
// memory.  head[warp] = SPH_NL_NONE marks a warp whose masks did not fit the pool.
#ifndef TILE_BULK_REPLAY
#define TILE_BULK_REPLAY 1
#endif

struct TileRecorder {
    NList nl; uint32_t prev_hdr; bool ok;
    __device__ __forceinline__ void init(const NList& n) { nl = n; prev_hdr = 0u; ok = n.pool != nullptr; }
    template <class WS>
    __device__ __forceinline__ void append(const WS& ws, int M, bool shifted, int warp_id, unsigned long long* counters) {
        if (!ok || M <= 0) return;
        const int lane = threadIdx.x & 31;
        const uint32_t rows = (uint32_t)M + 2u;
        uint32_t blk = 0;
        if (lane == 0) blk = atomicAdd(nl.used, rows) + 1u;
        blk = __shfl_sync(SPH_FULL_MASK, blk, 0);
        if ((unsigned long long)blk + rows > (unsigned long long)nl.pool_rows) {
            ok = false;                         // the warp's record is incomplete: the replaying pass searches again
            if (lane == 0) { nl.head[warp_id] = SPH_NL_NONE; atomicAdd(&counters[CNT_OVERFLOW], 1ull); }
            return;
        }
        __syncwarp();
        uint32_t* hdr = nl.pool + (size_t)blk * 32;
        hdr[lane] = lane == 0 ? 0u : (lane == 1 ? ((uint32_t)M | (shifted ? 0x100u : 0u)) : ws.hdr[lane]);
        hdr[32 + lane] = ws.bcode[lane];
        for (int m = 0; m < M; ++m) __stcs(hdr + (size_t)(m + 2) * 32 + lane, ws.mask[m][lane]);   // streaming: keep the state in L2
        if (lane == 0) { if (prev_hdr) nl.pool[(size_t)prev_hdr * 32] = blk; else nl.head[warp_id] = blk; }
        prev_hdr = blk;
    }
};

__device__ __forceinline__ uint32_t smem_addr(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

// drain(nz, shifted) is called once per recorded block with the header, shift codes and masks in ws
template <class WS, class Drain>
__device__ __forceinline__ void tile_replay(const GridDesc& g, const NList& nl, uint32_t blk, WS& ws, bool active, Drain&& drain) {
    const int lane = threadIdx.x & 31;
    constexpr int TILE_BLOCK_ROWS = WS::MMAX + 2;
#if TILE_BULK_REPLAY
    const uint32_t bar = smem_addr(&ws.bar), dst = smem_addr(ws.hdr);
    uint32_t phase = 0u;
    if (lane == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" :: "r"(bar));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncwarp();
#endif
    while (blk) {
        SPH_DBG_ASSERT((unsigned long long)blk + TILE_BLOCK_ROWS <= (unsigned long long)nl.pool_rows + TILE_BLOCK_ROWS, g);
        const uint32_t* src = nl.pool + (size_t)blk * 32;
        __syncwarp();                                                    // the previous block has been drained
#if TILE_BULK_REPLAY
        if (lane == 0) {     // one bulk copy of the whole block image (fixed size: a short block over-reads into the next rows of the pool)
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(bar), "r"((uint32_t)(TILE_BLOCK_ROWS * 128)) : "memory");
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                         :: "r"(dst), "l"(src), "r"((uint32_t)(TILE_BLOCK_ROWS * 128)), "r"(bar) : "memory");
        }
        uint32_t done = 0u;
        while (!done)
            asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                         : "=r"(done) : "r"(bar), "r"(phase) : "memory");
        phase ^= 1u;
#else
        ws.hdr[lane] = __ldcs(src + lane); ws.bcode[lane] = __ldcs(src + 32 + lane);
        __syncwarp();
        { const int M0 = (int)(ws.hdr[1] & 0xffu); for (int m = 0; m < M0; ++m) ws.mask[m][lane] = __ldcs(src + (size_t)(m + 2) * 32 + lane); }
#endif
        const uint32_t next = ws.hdr[0], w1 = ws.hdr[1];
        const int M = (int)(w1 & 0xffu);
        const bool shifted = (w1 & 0x100u) != 0u;
        SPH_DBG_ASSERT(blk < nl.pool_rows && M >= 1 && M <= WS::MMAX && (unsigned long long)blk + (unsigned)M + 2u <= nl.pool_rows, g);
        uint32_t nz = 0u;
        if (active)                                                      // a lane that is no destination of this pass drops its masks
            for (int m = 0; m < M; ++m) if (ws.mask[m][lane]) nz |= 0x80000000u >> m;
        drain(nz, shifted);
        blk = next;
    }
}

__device__ __forceinline__ unsigned long long warp_sum_u64(unsigned long long v) {
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(SPH_FULL_MASK, v, o);
    return v;
}
