// Pair-loop machinery shared by the density and acceleration kernels and the neighbour export.
//
// Mapping: one thread per destination particle in CELL-SORTED order, so a warp
// covers 1-3 x-adjacent cells and its lanes walk (almost) the same candidate runs: the 16-byte (x,y,z,h)
// loads of a warp hit 1-3 distinct addresses and are served as L1 broadcasts.
//
// Two phases per thread, both warp-synchronous:
//   phase 1  walk the 3^d neighbouring boxes (Fig.1) run by run; every candidate costs the
//            bit-specified predicate (R7) only; hits are appended to a per-thread queue in shared
//            memory (queue[t * BLOCK + tid]: conflict-free);
//   phase 2  when any lane's queue could overflow (and once at the end) the whole warp evaluates its queued
//            hits: the expensive body (kernel, EOS terms, viscosity) runs at ~mean/max neighbour-count lane
//            utilisation (~85 %) instead of the ~15 % hit rate of testing.
#pragma once
#include "sph_ctx.cuh"

#define PAIR_BLOCK 128
#define PAIR_QCAP 96
#define PAIR_CHUNK 32

// Walks all candidate runs of one destination particle.  Every lane of the warp must call this (inactive
// lanes pass active = false) because the run loops are warp-uniform and use warp votes.
template <int DIM, bool VARH, bool MERGED, class Policy>
__device__ __forceinline__ void walk_candidates(const GridDesc& g, const PairConsts& pc,
                                                const float4* __restrict__ posh,
                                                const uint32_t* __restrict__ cell_start,
                                                bool active, float4 pi, uint32_t ci, uint32_t my_mask,
                                                Policy& pol) {
    const int nc0 = g.nc[0], nc1 = g.nc[1], nc2 = g.nc[2], na = g.na;
    const int cx = (int)(ci % (uint32_t)nc0);
    const int t0 = (int)(ci / (uint32_t)nc0);
    const int cy = t0 % nc1, cz = t0 / nc1;
    const float cut2c = pair_cut2(pc.kh, pc.h_const, pc.h_const);

    auto segment = [&](bool ok, uint32_t s, uint32_t e, float sx, float sy, float sz) {
        const int len = ok ? (int)(e - s) : 0;
        const int maxlen = __reduce_max_sync(SPH_FULL_MASK, len);
        for (int c0 = 0; c0 < maxlen; c0 += PAIR_CHUNK) {
            pol.pre_chunk();
            const int lim = min(len, c0 + PAIR_CHUNK);
#pragma unroll 4
            for (int k = c0; k < lim; ++k) {
                const uint32_t j = s + (uint32_t)k;
                const float4 pj = __ldg(posh + j);
                const float dx = __fsub_rn(__fsub_rn(pi.x, pj.x), sx);
                const float dy = __fsub_rn(__fsub_rn(pi.y, pj.y), sy);
                float r2 = __fmaf_rn(dy, dy, __fmul_rn(dx, dx));
                if (DIM == 3) { const float dz = __fsub_rn(__fsub_rn(pi.z, pj.z), sz); r2 = __fmaf_rn(dz, dz, r2); }
                const float cut2 = VARH ? pair_cut2(pc.kh, pi.w, pj.w) : cut2c;
                if (r2 < cut2) pol.hit(j);
            }
        }
        pol.tested(len);
    };

    for (int oz = (DIM == 3 ? -1 : 0); oz <= (DIM == 3 ? 1 : 0); ++oz) {
        int z2 = cz + oz; float sz = 0.0f; bool okz = true;
        if (DIM == 3) {
            if (z2 < 0)         { if (g.per[2]) { z2 += nc2; sz = -g.L[2]; } else okz = false; }
            else if (z2 >= nc2) { if (g.per[2]) { z2 -= nc2; sz =  g.L[2]; } else okz = false; }
        }
        for (int oy = -1; oy <= 1; ++oy) {
            int y2 = cy + oy; float sy = 0.0f; bool oky = true;
            if (y2 < 0)         { if (g.per[1]) { y2 += nc1; sy = -g.L[1]; } else oky = false; }
            else if (y2 >= nc1) { if (g.per[1]) { y2 -= nc1; sy =  g.L[1]; } else oky = false; }
            const bool rowok = active && okz && oky;
            const uint32_t rowbase = rowok ? (uint32_t)((z2 * nc1 + y2) * nc0) : 0u;
            if (MERGED) {
                // all source arrays: the x-adjacent cells of a row are ONE contiguous run (key = x fastest)
                const int xlo = max(cx - 1, 0), xhi = min(cx + 1, nc0 - 1);
                uint32_t s = 0, e = 0;
                if (rowok) { s = cell_start[(rowbase + xlo) * na]; e = cell_start[(rowbase + xhi + 1) * na]; }
                segment(rowok, s, e, 0.0f, sy, sz);
                const bool wl = rowok && g.per[0] && cx == 0, wr = rowok && g.per[0] && cx == nc0 - 1;
                if (__any_sync(SPH_FULL_MASK, wl || wr)) {                    // the cell across the periodic seam
                    const int cw = wl ? nc0 - 1 : 0;
                    const float sx = wl ? -g.L[0] : g.L[0];
                    uint32_t s2 = 0, e2 = 0;
                    if (wl || wr) { s2 = cell_start[(rowbase + cw) * na]; e2 = cell_start[(rowbase + cw + 1) * na]; }
                    segment(wl || wr, s2, e2, sx, sy, sz);
                }
            } else {
                for (int ox = -1; ox <= 1; ++ox) {
                    int x2 = cx + ox; float sx = 0.0f; bool okx = true;
                    if (x2 < 0)         { if (g.per[0]) { x2 += nc0; sx = -g.L[0]; } else okx = false; }
                    else if (x2 >= nc0) { if (g.per[0]) { x2 -= nc0; sx =  g.L[0]; } else okx = false; }
                    for (int a = 0; a < na; ++a) {
                        const bool ok = rowok && okx && ((my_mask >> a) & 1u);
                        uint32_t s = 0, e = 0;
                        if (ok) { s = cell_start[(rowbase + x2) * na + a]; e = cell_start[(rowbase + x2) * na + a + 1]; }
                        if (__any_sync(SPH_FULL_MASK, ok)) segment(ok, s, e, sx, sy, sz);
                    }
                }
            }
        }
    }
}

// Minimum image for the FIELD arithmetic of phase 2 (any accurate image will do there; the set membership was
// decided bit-exactly in phase 1).  For a true neighbour |d_min| < L/3, so rint picks the same image as R7.
template <bool PER>
__device__ __forceinline__ float min_image(float d, float L, float invL) {
    if (PER) d = fmaf(-rintf(d * invL), L, d);
    return d;
}

// Queue + warp-synchronous flush shared by the density and acceleration policies (CRTP: Derived::body(j)).
template <class Derived>
struct QueuePolicy {
    uint32_t* q;               // shared memory, already offset by threadIdx.x
    int cnt;
    unsigned long long hits, tests;
    __device__ __forceinline__ void init(uint32_t* smem) { q = smem + threadIdx.x; cnt = 0; hits = 0; tests = 0; }
    __device__ __forceinline__ void hit(uint32_t j) { q[cnt * PAIR_BLOCK] = j; ++cnt; }
    __device__ __forceinline__ void tested(int len) { tests += (unsigned)len; }
    __device__ __forceinline__ void flush() {
        const int maxc = __reduce_max_sync(SPH_FULL_MASK, cnt);
#pragma unroll 2
        for (int t = 0; t < maxc; ++t)
            if (t < cnt) static_cast<Derived*>(this)->body(q[t * PAIR_BLOCK]);
        hits += (unsigned)cnt;
        cnt = 0;
    }
    __device__ __forceinline__ void pre_chunk() {
        if (__any_sync(SPH_FULL_MASK, cnt > PAIR_QCAP - PAIR_CHUNK)) flush();
    }
};

__device__ __forceinline__ unsigned long long warp_sum_u64(unsigned long long v) {
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(SPH_FULL_MASK, v, o);
    return v;
}
