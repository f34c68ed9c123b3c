// Pair-loop machinery shared by the density and acceleration kernels and the neighbour export.
//
// Mapping: one thread per destination particle in CELL-SORTED order, so the lanes
// of a warp sit in a few x-adjacent sub-cells and walk (almost) the same candidate runs: the 16-byte
// (x,y,z,h) loads of a warp hit a handful of addresses and are served as L1 broadcasts.
//
// Phase 1 (candidate tests).  For each of the 3^(d-1) stencil rows (Fig.1: the neighbouring
// boxes in y,z) the thread bounds the x-extent of its support sphere inside that row,
//     R_row = sqrt(R_i^2 - dy_min^2 - dz_min^2),   dy_min / dz_min = distance from the particle to the row's slab,
// and walks only the x sub-cells that intersect [x_i - R_row, x_i + R_row].  The bounds are conservative (they
// are widened by GridDesc::marg, and cell_coord is monotone in x), so no pair that passes the predicate is
// skipped; every candidate still takes the bit-specified predicate of DESIGN.md R7, which alone decides
// membership.  Hits are appended to a per-thread circular queue in shared memory (queue[slot * BLOCK + tid]:
// conflict-free).
// Phase 2 (evaluation).  When a lane's queue could overflow, and once at the end, the WHOLE warp drains T
// queued hits per lane: the expensive body (kernel, EOS terms, viscosity) runs at ~mean/max neighbour-count
// lane utilisation instead of the ~30 % hit rate of testing.  A recording policy also writes the drained rows
// (32 lanes x T, coalesced) to the neighbour-row pool for the acceleration pass to replay.
#pragma once
#include "sph_ctx.cuh"
#include <type_traits>

#define PAIR_BLOCK 128
#ifndef PAIR_QCAP
#define PAIR_QCAP 64              // queue slots per thread, power of two
#endif
#ifndef PAIR_CHUNK
#define PAIR_CHUNK 16             // candidates tested between two queue-level checks
#endif
#ifndef PAIR_MIN_DRAIN
#define PAIR_MIN_DRAIN 16
#endif
#define PAIR_QSTRIDE (PAIR_BLOCK * 4u)                 // bytes between two slots of one thread
#define PAIR_QBYTES_MASK (PAIR_QCAP * PAIR_QSTRIDE - 1u)

__device__ __forceinline__ void sts_u32(uint32_t saddr, uint32_t v) { asm volatile("st.shared.u32 [%0], %1;" :: "r"(saddr), "r"(v) : "memory"); }
__device__ __forceinline__ uint32_t lds_u32(uint32_t saddr) { uint32_t v; asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(saddr) : "memory"); return v; }

// Walks all candidate runs of one destination particle.  Every lane of the warp must call this (inactive
// lanes pass active = false) because the run loops are warp-uniform and use warp votes.
template <int DIM, bool VARH, class Policy>
__device__ __forceinline__ void walk_candidates(const GridDesc& g, const PairConsts& pc,
                                                const float4* __restrict__ posh,
                                                const uint32_t* __restrict__ cell_start,
                                                bool active, float4 pi, uint32_t ci, Policy& pol) {
    const int nc0 = g.nc[0], nc1 = g.nc[1], nc2 = g.nc[2], na = g.na;
    const int t0 = (int)(ci / (uint32_t)nc0);
    const int cy = t0 % nc1, cz = t0 / nc1;
    const float cut2c = pair_cut2(pc.kh, pc.h_const, pc.h_const);
    // largest cut-off any pair of particle i can have: k (h_i + h_max) / 2, widened by 1e-5
    const float R = pc.kh * (VARH ? (pi.w + pc.h_const) : (pc.h_const + pc.h_const)) * 1.00001f;
    const float R2 = R * R;
    const float fy = pi.y - fmaf((float)cy, g.cell[1], g.lo[1]);          // position inside the own cell
    const float fz = DIM == 3 ? pi.z - fmaf((float)cz, g.cell[2], g.lo[2]) : 0.0f;

    // one contiguous run [s, e) of the sorted order, tested against particle i with image shift (sx, sy, sz)
    auto segment = [&](auto shift_tag, bool ok, uint32_t s, uint32_t e, float sx, float sy, float sz) {
        constexpr bool SHIFT = decltype(shift_tag)::value;
        const int len = ok ? (int)(e - s) : 0;
        const int maxlen = __reduce_max_sync(SPH_FULL_MASK, len);
        for (int c0 = 0; c0 < maxlen; c0 += PAIR_CHUNK) {
            pol.pre_chunk();
            const int lim = min(len, c0 + PAIR_CHUNK);
#pragma unroll 4
            for (int k = c0; k < lim; ++k) {
                const uint32_t j = s + (uint32_t)k;
                const float4 pj = __ldg(posh + j);
                float dx = __fsub_rn(pi.x, pj.x), dy = __fsub_rn(pi.y, pj.y);
                if (SHIFT) { dx = __fsub_rn(dx, sx); dy = __fsub_rn(dy, sy); }
                float r2 = __fmaf_rn(dy, dy, __fmul_rn(dx, dx));
                if (DIM == 3) {
                    float dz = __fsub_rn(pi.z, pj.z);
                    if (SHIFT) dz = __fsub_rn(dz, sz);
                    r2 = __fmaf_rn(dz, dz, r2);
                }
                const float cut2 = VARH ? pair_cut2(pc.kh, pi.w, pj.w) : cut2c;
                if (r2 < cut2) pol.hit(j);
            }
        }
        pol.tested(len);
    };

    for (int oz = (DIM == 3 ? -1 : 0); oz <= (DIM == 3 ? 1 : 0); ++oz) {
        int z2 = cz + oz; float sz = 0.0f; bool okz = true; float dzm = 0.0f;
        if (DIM == 3) {
            if (z2 < 0)         { if (g.per[2]) { z2 += nc2; sz = -g.L[2]; } else okz = false; }
            else if (z2 >= nc2) { if (g.per[2]) { z2 -= nc2; sz =  g.L[2]; } else okz = false; }
            dzm = oz < 0 ? fz : (oz > 0 ? g.cell[2] - fz : 0.0f);
            dzm = fmaxf(dzm - g.marg[2], 0.0f);
        }
        for (int oy = -1; oy <= 1; ++oy) {
            int y2 = cy + oy; float sy = 0.0f; bool oky = true;
            if (y2 < 0)         { if (g.per[1]) { y2 += nc1; sy = -g.L[1]; } else oky = false; }
            else if (y2 >= nc1) { if (g.per[1]) { y2 -= nc1; sy =  g.L[1]; } else oky = false; }
            float dym = oy < 0 ? fy : (oy > 0 ? g.cell[1] - fy : 0.0f);
            dym = fmaxf(dym - g.marg[1], 0.0f);
            const float rem = R2 - dym * dym - dzm * dzm;
            const bool rowok = active && okz && oky && rem > 0.0f;
            const uint32_t rowbase = rowok ? (uint32_t)((z2 * nc1 + y2) * nc0) : 0u;
            const float Rrow = sqrtf(fmaxf(rem, 0.0f)) + g.marg[0];
            const int cl = __float2int_rd((pi.x - Rrow - g.lo[0]) * g.inv_cell[0]);
            const int ch = __float2int_rd((pi.x + Rrow - g.lo[0]) * g.inv_cell[0]);
            const int a = max(cl, 0), b = min(ch, nc0 - 1);
            const bool shifted_row = (sy != 0.0f) || (sz != 0.0f);
            {   // the sub-cells inside the box
                const bool ok = rowok && a <= b;
                uint32_t s = 0, e = 0;
                if (ok) { s = cell_start[(rowbase + a) * na]; e = cell_start[(rowbase + b + 1) * na]; }
                if (__any_sync(SPH_FULL_MASK, ok && shifted_row)) segment(std::true_type{}, ok, s, e, 0.0f, sy, sz);
                else segment(std::false_type{}, ok, s, e, 0.0f, sy, sz);
            }
            if (g.per[0]) {   // the parts of the interval across the periodic seam (one slack sub-cell each,
                              // never overlapping the run above)
                const bool wl = rowok && cl < 0, wr = rowok && ch >= nc0;
                if (__any_sync(SPH_FULL_MASK, wl)) {
                    const int a2 = max(cl + nc0 - 1, b + 1);
                    const bool ok = wl && a2 <= nc0 - 1;
                    uint32_t s = 0, e = 0;
                    if (ok) { s = cell_start[(rowbase + a2) * na]; e = cell_start[(rowbase + nc0) * na]; }
                    segment(std::true_type{}, ok, s, e, -g.L[0], sy, sz);
                }
                if (__any_sync(SPH_FULL_MASK, wr)) {
                    const int b2 = min(ch - nc0 + 1, a - 1);
                    const bool ok = wr && b2 >= 0;
                    uint32_t s = 0, e = 0;
                    if (ok) { s = cell_start[rowbase * na]; e = cell_start[(rowbase + b2 + 1) * na]; }
                    segment(std::true_type{}, ok, s, e, g.L[0], sy, sz);
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

// Circular hit queue + warp-synchronous drain shared by the density and acceleration policies
// (CRTP: Derived::body(j)).  FILTER: the walker visits the runs of ALL arrays (key = cell * na + array keeps
// them contiguous); a destination whose source mask is not "all arrays" drops hits from the other arrays here.
// RECORD: drained rows are appended to the neighbour-row pool.
template <class Derived, bool FILTER, bool RECORD>
struct QueuePolicy {
    uint32_t qaddr;            // shared-space address of this thread's slot 0
    uint32_t rpos, wpos;       // byte offsets (multiples of PAIR_QSTRIDE, unmasked) of the read / write slot
    int cnt;
    bool is_active;
    unsigned long long hits, tests;
    const uint32_t* meta; uint32_t src_mask;      // FILTER
    NList nl; uint32_t prev_hdr; bool rec_ok; unsigned long long* counters;   // RECORD

    __device__ __forceinline__ void init(uint32_t* smem, bool active, const uint32_t* meta_, uint32_t mask_) {
        qaddr = (uint32_t)__cvta_generic_to_shared(smem + threadIdx.x); rpos = 0; wpos = 0; cnt = 0;
        hits = 0; tests = 0; is_active = active;
        meta = meta_; src_mask = mask_; prev_hdr = 0; rec_ok = RECORD; counters = nullptr;
    }
    __device__ __forceinline__ void hit(uint32_t j) {
        if (FILTER) { if (!((src_mask >> (__ldg(meta + j) >> SPH_META_IDX_BITS)) & 1u)) return; }
        sts_u32(qaddr + (wpos & PAIR_QBYTES_MASK), j); wpos += PAIR_QSTRIDE; ++cnt;
    }
    __device__ __forceinline__ void tested(int len) { tests += (unsigned)len; }

    // drains T rows (lanes with fewer queued hits contribute SPH_NL_NONE)
    __device__ __forceinline__ void drain(int T) {
        if (T <= 0) return;
        const int lane = threadIdx.x & 31;
        size_t row0 = 0;
        if (RECORD && rec_ok) {
            uint32_t base = 0;
            if (lane == 0) base = atomicAdd(nl.used, (uint32_t)T + 1u) + 1u;
            base = __shfl_sync(SPH_FULL_MASK, base, 0);
            if ((unsigned long long)base + (unsigned)T + 1ull > (unsigned long long)nl.pool_rows) {
                rec_ok = false;
                if (lane == 0) atomicAdd(&counters[CNT_OVERFLOW], 1ull);
            } else {
                if (lane == 0) {
                    if (prev_hdr) nl.pool[(size_t)prev_hdr * 32] = base;
                    else nl.head[(blockIdx.x * PAIR_BLOCK + threadIdx.x) >> 5] = base;
                    nl.pool[(size_t)base * 32] = 0u; nl.pool[(size_t)base * 32 + 1] = (uint32_t)T;
                }
                prev_hdr = base;
                row0 = ((size_t)base + 1) * 32 + lane;
            }
        }
        const int mine = min(T, cnt);
#pragma unroll 2
        for (int t = 0; t < T; ++t) {
            uint32_t j = SPH_NL_NONE;
            if (t < mine) { j = lds_u32(qaddr + ((rpos + (uint32_t)t * PAIR_QSTRIDE) & PAIR_QBYTES_MASK)); static_cast<Derived*>(this)->body(j); }
            if (RECORD && rec_ok) nl.pool[row0 + (size_t)t * 32] = j;
        }
        hits += (unsigned)mine;
        rpos += (uint32_t)mine * PAIR_QSTRIDE; cnt -= mine;
    }
    __device__ __forceinline__ void pre_chunk() {
        const int maxc = __reduce_max_sync(SPH_FULL_MASK, cnt);
        if (maxc > PAIR_QCAP - PAIR_CHUNK) {
            const int minc = __reduce_min_sync(SPH_FULL_MASK, is_active ? cnt : 0x7fffffff);
            drain(max(max(min(minc, maxc), maxc - (PAIR_QCAP - PAIR_CHUNK)), min(PAIR_MIN_DRAIN, maxc)));
        }
    }
    __device__ __forceinline__ void flush() { drain(__reduce_max_sync(SPH_FULL_MASK, cnt)); }
};

__device__ __forceinline__ unsigned long long warp_sum_u64(unsigned long long v) {
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(SPH_FULL_MASK, v, o);
    return v;
}
