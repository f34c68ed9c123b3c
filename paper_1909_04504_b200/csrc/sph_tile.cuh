// Warp-tile pair machinery: candidate tests, hit masks, drain, mask records.
//
// Mapping.  A warp owns 32 consecutive particles of the CELL-SORTED order (x sub-cell fastest), i.e. a short
// tube along x inside one stencil row (Fig.1).  For each of the 3^(d-1) neighbouring rows the
// warp's candidates are ONE contiguous run of the sorted order: the sub-cells [sub_lo - xsub, sub_hi + xsub]
// (a coarse cell = xsub sub-cells >= the support radius, so nothing closer than the cut-off lies outside).
//
// Phase 1 (tests).  The run is read once, coalesced, 32 candidates at a time, and staged as SoA in shared
// memory; every lane then tests ITS particle against the SAME candidate, read as a shared-memory broadcast
// (no divergent loads, no bank conflicts), four candidates per step with packed f32x2 arithmetic (FADD2 /
// FMUL2 / FFMA2, sm_100).  The arithmetic is the bit-specified predicate of DESIGN.md R7; rounding of the
// packed forms is the same round-to-nearest as the scalar forms.  The result is one 32-bit hit mask per lane
// and batch, stored to shared memory (mask[m][lane]) with the batch's first sorted index (base[m]).
// Phase 2 (evaluation).  When the mask store is full, and once at the end, the warp drains it: every lane pops
// its own hits in order and runs the expensive body (kernel, EOS terms, viscosity) on them, so the body runs
// at mean/max neighbour-count lane utilisation instead of the hit rate of the tests.
// Records.  A recording pass also copies the masks and bases (not the hit indices: 4 B per 32 tests instead of
// 4 B per hit) to the record pool; the acceleration pass of the same evaluation replays them (tile_replay)
// and tests nothing.
#pragma once
#include "sph_ctx.cuh"
#include <type_traits>

#define TILE_BLOCK 128
#define TILE_WARPS (TILE_BLOCK / 32)
#ifndef TILE_MIN_BLOCKS
#define TILE_MIN_BLOCKS 8                 // resident blocks per SM the pair kernels are compiled for (64 registers)
#endif
#ifndef TILE_MIN_BLOCKS_ACCEL
#define TILE_MIN_BLOCKS_ACCEL 6           // the momentum kernel is 3-8 % faster with 80 registers and 6 blocks (measured, C3, C4)
#endif
#ifndef TILE_DRAIN_DEPTH_REPLAY
#define TILE_DRAIN_DEPTH_REPLAY 3         // hits in flight in the replaying momentum kernel (-4 % on C3; the searching kernels lose with 3)
#endif
#ifndef TILE_DRAIN_DEPTH_DENSITY
#define TILE_DRAIN_DEPTH_DENSITY 3         // hits in flight in the density drain (3: -2 % on C3; 4 is no better)
#endif
#ifndef TILE_MMAX
#define TILE_MMAX 30                       // masks per warp before a forced drain (<= 30: 30 bases + 2 words = one header row)
#endif

struct __align__(16) TileWarpSmem {
    float x[32], y[32], z[32], h[32];      // one staged batch of candidates, SoA
    uint32_t mask[TILE_MMAX][32];          // hit masks, [batch][lane]
    uint32_t base[32];                     // first sorted index of every batch
    uint32_t seg_s[32], seg_e[32], seg_c[32];   // candidate runs of the current group: [s, e) and image-shift code
};

struct TileState {
    int M;                                 // masks stored since the last drain (warp-uniform)
    uint32_t nz;                           // bit m: this lane's mask m has hits
    bool shifted;                          // some stored batch came from a periodic image (warp-uniform)
    unsigned long long tests;              // predicate evaluations of this lane's particle
    unsigned long long hits;               // predicate hits of this lane's particle
    __device__ __forceinline__ void reset() { M = 0; nz = 0u; shifted = false; }
};

__device__ __forceinline__ float2 f2(float a, float b) { return make_float2(a, b); }
__device__ __forceinline__ float2 sub2(float2 a, float2 b) { return __fadd2_rn(a, f2(-b.x, -b.y)); }

// Predicate of DESIGN.md R7 for 4 staged candidates c..c+3 against this lane's particle: bit k of the result
// is the hit of candidate c+k.   d = fl(fl(x_i - x_j) - shift);  r2 = fma(dz,dz,fma(dy,dy,fl(dx*dx)));
// cut = fl(kh * fl(h_i + h_j));  hit <=> r2 < fl(cut*cut).
template <int DIM, bool VARH, bool SHIFT>
__device__ __forceinline__ uint32_t tile_test4(const TileWarpSmem& ws, int c, float2 xi, float2 yi, float2 zi,
                                               float2 sx, float2 sy, float2 sz, float2 cut2c, float2 kh2, float2 hi2) {
    const float4 X = *reinterpret_cast<const float4*>(ws.x + c);
    const float4 Y = *reinterpret_cast<const float4*>(ws.y + c);
    float2 dxa = sub2(xi, f2(X.x, X.y)), dxb = sub2(xi, f2(X.z, X.w));
    float2 dya = sub2(yi, f2(Y.x, Y.y)), dyb = sub2(yi, f2(Y.z, Y.w));
    if (SHIFT) { dxa = sub2(dxa, sx); dxb = sub2(dxb, sx); dya = sub2(dya, sy); dyb = sub2(dyb, sy); }
    float2 ra = __ffma2_rn(dya, dya, __fmul2_rn(dxa, dxa));
    float2 rb = __ffma2_rn(dyb, dyb, __fmul2_rn(dxb, dxb));
    if (DIM == 3) {
        const float4 Z = *reinterpret_cast<const float4*>(ws.z + c);
        float2 dza = sub2(zi, f2(Z.x, Z.y)), dzb = sub2(zi, f2(Z.z, Z.w));
        if (SHIFT) { dza = sub2(dza, sz); dzb = sub2(dzb, sz); }
        ra = __ffma2_rn(dza, dza, ra); rb = __ffma2_rn(dzb, dzb, rb);
    }
    float2 ca = cut2c, cb = cut2c;
    if (VARH) {
        const float4 H = *reinterpret_cast<const float4*>(ws.h + c);
        const float2 ta = __fmul2_rn(kh2, __fadd2_rn(hi2, f2(H.x, H.y)));
        const float2 tb = __fmul2_rn(kh2, __fadd2_rn(hi2, f2(H.z, H.w)));
        ca = __fmul2_rn(ta, ta); cb = __fmul2_rn(tb, tb);
    }
    uint32_t m = 0;
    if (ra.x < ca.x) m |= 1u;
    if (ra.y < ca.y) m |= 2u;
    if (rb.x < cb.x) m |= 4u;
    if (rb.y < cb.y) m |= 8u;
    return m;
}

// Walks every candidate run of the warp's 32 particles.  `drain()` is called (warp-uniformly, from ONE site)
// whenever the mask store holds TILE_MMAX batches, and once at the end; it must consume the masks and call
// st.reset().  All 32 lanes must call this.
//   row = cell / nc0 (the stencil row of the particle), sub = cell % nc0 (its x sub-cell), -1 / 0 for lanes
//   past the end of the sorted order.
// Structure: for every GROUP of lanes (below) the 3^(d-1) x 3 candidate runs (stencil row x {inside the box,
// image across the low x seam, image across the high x seam}) are looked up by 27 lanes in parallel and
// written to a small table; one flat loop then streams the runs batch by batch.
template <int DIM, bool VARH, class Drain>
__device__ __forceinline__ void tile_walk(const GridDesc& g, const PairConsts& pc,
                                          const float4* __restrict__ posh, const uint32_t* __restrict__ cell_start,
                                          bool active, float4 pi, int row, int sub,
                                          TileWarpSmem& ws, TileState& st, Drain&& drain) {
    const int lane = threadIdx.x & 31;
    const int nc0 = g.nc[0], nc1 = g.nc[1], nc2 = g.nc[2], na = g.na, xsub = g.xsub;
    const float2 xi = f2(pi.x, pi.x), yi = f2(pi.y, pi.y), zi = f2(pi.z, pi.z);
    const float2 kh2 = f2(pc.kh, pc.kh), hi2 = f2(pi.w, pi.w);
    const float cc = pair_cut2(pc.kh, pc.h_const, pc.h_const);
    const float2 cut2c = f2(cc, cc);
    constexpr int NSEG = (DIM == 3 ? 27 : 9);

    // groups: maximal lane ranges of one stencil row without an x gap wider than two coarse cells (a wider
    // gap means the windows of its two sides are disjoint, so splitting there saves tests)
    const int prow = __shfl_up_sync(SPH_FULL_MASK, row, 1), psub = __shfl_up_sync(SPH_FULL_MASK, sub, 1);
    const bool brk = lane == 0 || row != prow || sub - psub > 2 * xsub;
    const unsigned brkmask = __ballot_sync(SPH_FULL_MASK, brk);
    unsigned remaining = __ballot_sync(SPH_FULL_MASK, active);

    bool ing = false, done = false, seg_shift = false;
    int seg = NSEG;                                   // forces the first group set-up
    uint32_t b0 = 0u, e = 0u;
    unsigned segs = 0u;                               // non-empty runs of the current group still to stream
    float2 sx = f2(0.0f, 0.0f), sy = sx, sz = sx;

    while (!done) {
        while (st.M < TILE_MMAX) {
            if (b0 >= e) {
                if (++seg >= NSEG) {                  // next group
                    if (!remaining) { done = true; break; }
                    const int leader = __ffs(remaining) - 1;
                    const int gs = 31 - __clz(brkmask & (0xffffffffu >> (31 - leader)));      // start of the leader's range
                    const unsigned above = leader < 31 ? (brkmask & (0xffffffffu << (leader + 1))) : 0u;
                    const int ge = above ? __ffs(above) - 1 : 32;                               // one past its end
                    const unsigned range = (ge == 32 ? 0xffffffffu : ((1u << ge) - 1u)) & (0xffffffffu << gs);
                    const unsigned gmask = remaining & range;
                    remaining &= ~gmask;
                    ing = (gmask >> lane) & 1u;
                    const int first = __ffs(gmask) - 1, last = 31 - __clz(gmask);
                    const int grow = __shfl_sync(SPH_FULL_MASK, row, first);
                    const int sub_lo = __shfl_sync(SPH_FULL_MASK, sub, first), sub_hi = __shfl_sync(SPH_FULL_MASK, sub, last);
                    const int cy = grow % nc1, cz = grow / nc1;
                    // x reach in sub-cells: a pair of the group is closer than R = k (h_group_max + h_max) / 2, so
                    // its sub-cell indices differ by at most floor(R / sub-cell) + 1 (<= xsub: cell >= k h_max)
                    int nx = xsub;
                    if (VARH) {
                        const float hg = __uint_as_float(__reduce_max_sync(SPH_FULL_MASK, ing ? __float_as_uint(pi.w) : 0u));
                        const float R = pc.kh * (hg + pc.h_const) * 1.0001f;
                        nx = min(xsub, __float2int_rd(R * g.inv_cell[0]) + 1);
                    }
                    const int a = sub_lo - nx, b = sub_hi + nx;
                    __syncwarp();
                    bool nonempty = false;
                    if (lane < NSEG) {                // lane = 9 (oz+1) + 3 (oy+1) + part
                        const int part = lane % 3, oy = (lane / 3) % 3 - 1, oz = DIM == 3 ? lane / 9 - 1 : 0;
                        int y2 = cy + oy, z2 = cz + oz; uint32_t code = 0u; bool ok = true;
                        if (y2 < 0)         { if (g.per[1]) { y2 += nc1; code |= 1u << 2; } else ok = false; }
                        else if (y2 >= nc1) { if (g.per[1]) { y2 -= nc1; code |= 2u << 2; } else ok = false; }
                        if (z2 < 0)         { if (g.per[2]) { z2 += nc2; code |= 1u << 4; } else ok = false; }
                        else if (z2 >= nc2) { if (g.per[2]) { z2 -= nc2; code |= 2u << 4; } else ok = false; }
                        int c0, c1;
                        if (part == 0)      { c0 = max(a, 0); c1 = min(b, nc0 - 1); }
                        else if (part == 1) { c0 = a + nc0; c1 = nc0 - 1; code |= 1u; ok = ok && g.per[0] && a < 0; }
                        else                { c0 = 0; c1 = b - nc0; code |= 2u; ok = ok && g.per[0] && b >= nc0; }
                        uint32_t s_ = 0u, e_ = 0u;
                        if (ok) {
                            const uint32_t rowbase = (uint32_t)((z2 * nc1 + y2) * nc0);
                            s_ = __ldg(cell_start + (size_t)(rowbase + (uint32_t)c0) * na);
                            e_ = __ldg(cell_start + (size_t)(rowbase + (uint32_t)c1 + 1u) * na);
                        }
                        ws.seg_s[lane] = s_; ws.seg_e[lane] = e_; ws.seg_c[lane] = code;
                        nonempty = s_ < e_;
                    }
                    segs = __ballot_sync(SPH_FULL_MASK, nonempty);      // runs that hold candidates
                    __syncwarp();
                    seg = -1; b0 = e = 0u;
                    continue;
                }
                if (segs == 0u) { seg = NSEG; b0 = e = 0u; continue; }   // group done
                seg = __ffs(segs) - 1; segs &= segs - 1u;
                b0 = ws.seg_s[seg]; e = ws.seg_e[seg];
                const uint32_t code = ws.seg_c[seg];      // image shifts: 1 -> -L (wrapped below), 2 -> +L (wrapped above)
                seg_shift = code != 0u;
                const float fx = (code & 3u) == 1u ? -g.L[0] : ((code & 3u) == 2u ? g.L[0] : 0.0f);
                const float fy = ((code >> 2) & 3u) == 1u ? -g.L[1] : (((code >> 2) & 3u) == 2u ? g.L[1] : 0.0f);
                const float fz = ((code >> 4) & 3u) == 1u ? -g.L[2] : (((code >> 4) & 3u) == 2u ? g.L[2] : 0.0f);
                sx = f2(fx, fx); sy = f2(fy, fy); sz = f2(fz, fz);
                continue;
            }
            // one batch of <= 32 candidates [b0, min(b0 + 32, e))
            const uint32_t j = b0 + (uint32_t)lane;
            float4 pj = make_float4(3.0e38f, 0.0f, 0.0f, 0.0f);           // padding: r2 = inf, never a hit
            if (j < e) pj = __ldg(posh + j);
            __syncwarp();                                                  // readers of the previous batch are done
            ws.x[lane] = pj.x; ws.y[lane] = pj.y;
            if (DIM == 3) ws.z[lane] = pj.z;
            if (VARH) ws.h[lane] = pj.w;
            __syncwarp();
            const int len = (int)min(32u, e - b0);
            const int n8 = (len + 7) >> 3;                                // 8 candidates per branch-free step
            uint32_t mask = 0;
            if (seg_shift) {
#pragma unroll
                for (int u = 0; u < 4; ++u)
                    if (u < n8) {
                        const uint32_t m0 = tile_test4<DIM, VARH, true>(ws, 8 * u, xi, yi, zi, sx, sy, sz, cut2c, kh2, hi2);
                        const uint32_t m1 = tile_test4<DIM, VARH, true>(ws, 8 * u + 4, xi, yi, zi, sx, sy, sz, cut2c, kh2, hi2);
                        mask |= (m0 << (8 * u)) | (m1 << (8 * u + 4));
                    }
                st.shifted = true;
            } else {
#pragma unroll
                for (int u = 0; u < 4; ++u)
                    if (u < n8) {
                        const uint32_t m0 = tile_test4<DIM, VARH, false>(ws, 8 * u, xi, yi, zi, sx, sy, sz, cut2c, kh2, hi2);
                        const uint32_t m1 = tile_test4<DIM, VARH, false>(ws, 8 * u + 4, xi, yi, zi, sx, sy, sz, cut2c, kh2, hi2);
                        mask |= (m0 << (8 * u)) | (m1 << (8 * u + 4));
                    }
            }
            if (!ing) mask = 0u;
            ws.mask[st.M][lane] = mask;
            if (mask) st.nz |= 1u << st.M;
            if (lane == 0) ws.base[st.M] = b0;
            if (ing) st.tests += (unsigned)len;
            st.hits += (unsigned)__popc(mask);
            ++st.M;
            b0 += 32u;
        }
        drain();                                                           // consumes the masks, resets st
    }
}

// Every lane pops its own hits of the stored batches in order (nz: the lane's non-empty masks) and evaluates
// them.  Branch-free and software-pipelined: DEPTH hits are in flight, the source data of a later hit is
// gathered (Src = load(sorted index)) before the current one is computed, so the gather latency (L2: the sorted
// state does not fit L1) overlaps the arithmetic.  A lane that has run out keeps executing with has = false and
// the harmless index `idle` (its own particle) until the slowest lane of the warp is done; compute(src, has)
// must contribute nothing when has is false.
template <class Src, int DEPTH = 2, class Load, class Compute>
__device__ __forceinline__ void tile_drain(TileWarpSmem& ws, uint32_t nz, uint32_t idle, Load&& load, Compute&& compute) {
    const int lane = threadIdx.x & 31;
    __syncwarp();
    uint32_t cur = 0u, b = 0u;
    auto pop = [&](bool& has) -> uint32_t {
        const bool refill = cur == 0u && nz != 0u;
        const int m = max(__ffs(nz) - 1, 0);
        const uint32_t nm = ws.mask[m][lane], nb = ws.base[m];
        cur = refill ? nm : cur; b = refill ? nb : b; nz = refill ? (nz & (nz - 1u)) : nz;
        has = cur != 0u;
        const uint32_t j = has ? b + (uint32_t)(__ffs(cur) - 1) : idle;
        cur &= cur - 1u;                        // stays 0 when it is 0
        return j;
    };
    Src R[DEPTH]; bool H[DEPTH];                    // DEPTH hits in flight; fully unrolled, so R and H live in registers
#pragma unroll
    for (int d = 0; d + 1 < DEPTH; ++d) R[d] = load(pop(H[d]));
    for (;;) {
#pragma unroll
        for (int d = 0; d < DEPTH; ++d) {
            const int nx = (d + DEPTH - 1) % DEPTH;
            R[nx] = load(pop(H[nx]));               // gather for a later hit ...
            compute(R[d], H[d]);                    // ... while this one is evaluated
        }
        if (!__any_sync(SPH_FULL_MASK, H[0])) break;   // pops are in order: no pending hit 0 means no pending hit at all
    }
    __syncwarp();
}

// ---- mask records (recorded by the density pass, replayed by the acceleration pass) -----------------------
// The pool is an array of ROWS of 32 words.  A warp appends BLOCKS: a header row {next block (row index, 0 =
// end), number of batches M <= TILE_MMAX | 0x100 if a batch came from a periodic image, base[0..M-1]} followed
// by M rows of masks (word = lane).  head[warp] = SPH_NL_NONE marks a warp whose masks did not fit the pool.
struct TileRecorder {
    NList nl; uint32_t prev_hdr; bool ok;
    __device__ __forceinline__ void init(const NList& n) { nl = n; prev_hdr = 0u; ok = n.pool != nullptr; }
    __device__ __forceinline__ void append(const TileWarpSmem& ws, int M, bool shifted, int warp_id, unsigned long long* counters) {
        if (!ok || M <= 0) return;
        const int lane = threadIdx.x & 31;
        uint32_t blk = 0;
        if (lane == 0) blk = atomicAdd(nl.used, (uint32_t)M + 1u) + 1u;
        blk = __shfl_sync(SPH_FULL_MASK, blk, 0);
        if ((unsigned long long)blk + (unsigned)M + 1ull > (unsigned long long)nl.pool_rows) {
            ok = false;                         // the warp's record is incomplete: the replaying pass searches again
            if (lane == 0) { nl.head[warp_id] = SPH_NL_NONE; atomicAdd(&counters[CNT_OVERFLOW], 1ull); }
            return;
        }
        __syncwarp();
        uint32_t* hdr = nl.pool + (size_t)blk * 32;
        hdr[lane] = lane == 0 ? 0u : (lane == 1 ? ((uint32_t)M | (shifted ? 0x100u : 0u)) : ws.base[lane - 2]);
        for (int m = 0; m < M; ++m) __stcs(hdr + (size_t)(m + 1) * 32 + lane, ws.mask[m][lane]);   // streaming: keep the state in L2
        if (lane == 0) { if (prev_hdr) nl.pool[(size_t)prev_hdr * 32] = blk; else nl.head[warp_id] = blk; }
        prev_hdr = blk;
    }
};

// drain(nz, shifted) is called once per recorded block with the masks and bases in ws
template <class Drain>
__device__ __forceinline__ void tile_replay(const NList& nl, uint32_t blk, TileWarpSmem& ws, bool active, unsigned long long& hits, Drain&& drain) {
    const int lane = threadIdx.x & 31;
    while (blk) {
        const uint32_t* hdr = nl.pool + (size_t)blk * 32;
        const uint32_t hw = __ldcs(hdr + lane);
        const uint32_t next = __shfl_sync(SPH_FULL_MASK, hw, 0);
        const uint32_t w1 = __shfl_sync(SPH_FULL_MASK, hw, 1);
        const int M = (int)(w1 & 0xffu);
        __syncwarp();
        if (lane >= 2) ws.base[lane - 2] = hw;
        uint32_t nz = 0u;
        for (int m0 = 0; m0 < M; m0 += 8) {                              // 8 independent loads in flight
            uint32_t w[8];
#pragma unroll
            for (int k = 0; k < 8; ++k) w[k] = (m0 + k < M && active) ? __ldcs(hdr + (size_t)(m0 + k + 1) * 32 + lane) : 0u;   // a lane that is no destination of this pass drops its masks
#pragma unroll
            for (int k = 0; k < 8; ++k) if (m0 + k < M) { ws.mask[m0 + k][lane] = w[k]; if (w[k]) nz |= 1u << (m0 + k); hits += (unsigned)__popc(w[k]); }
        }
        drain(nz, (w1 & 0x100u) != 0u);
        blk = next;
    }
}

__device__ __forceinline__ unsigned long long warp_sum_u64(unsigned long long v) {
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(SPH_FULL_MASK, v, o);
    return v;
}

// Minimum image for the FIELD arithmetic of phase 2 (any accurate image will do there; the set membership was
// decided bit-exactly in phase 1).  For a true neighbour |d_min| < L/3, so rint picks the same image as R7.
__device__ __forceinline__ float min_image(float d, float L, float invL) { return fmaf(-rintf(d * invL), L, d); }
