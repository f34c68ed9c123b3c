// NNPS build (Sec.2.2): cell key -> counting sort by key -> cell-start offsets -> gather of
// every property into cell order; the fused predictor-corrector update (eqs. 12-14) that feeds it;
// the caller-order output gathers; and the neighbour-list export used for the bit-exact set parity.
// All of these stream each particle once: they are HBM-bandwidth kernels.
#include "sph_tile.cuh"

#define NB 256

// ------------------------------------------------------------------------------------------------
// cell of a position (a1).  Linear key, x fastest, so the 3 x-adjacent cells of a stencil row are one run.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t cell_of(const GridDesc& g, float4 p, int level, bool& oob) {   // float-rounded position: the search runs in float
    const LevelDesc& Lv = g.lev[level];
    int c[3]; const float x[3] = { p.x, p.y, p.z };
    oob = false;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        if (a < g.dim) {
            if (!(x[a] >= g.lo[a] && x[a] <= g.hi[a])) oob = true;   // also catches NaN; periodic axes too:
                                                                      // the caller's positions must lie in the box
            c[a] = cell_coord(x[a], g.lo[a], Lv.inv_cell[a], Lv.nc[a]);
        } else c[a] = 0;
    }
    return Lv.base + (uint32_t)((c[2] * Lv.nc[1] + c[1]) * Lv.nc[0] + c[0]);
}

// positive reals order like their bit patterns: min/max through integer atomics
#ifdef SPH_REAL_DOUBLE
typedef long long real_bits;
__device__ __forceinline__ real_bits real_as_bits(double x) { return __double_as_longlong(x); }
#else
typedef int real_bits;
__device__ __forceinline__ real_bits real_as_bits(float x) { return __float_as_int(x); }
#endif
__device__ __forceinline__ real_bits shfl_xor_bits(real_bits v, int o) { return __shfl_xor_sync(SPH_FULL_MASK, v, o); }

// Loads the caller's SoA arrays into the (not yet sorted) real4 groups and reduces h_min / h_max, |m|_min / |m|_max.
__global__ void __launch_bounds__(NB)
k_pack(PackArgs A, SortedState S, int n, PairConsts pc, real_bits* __restrict__ hminmax) {
    const int gidx = blockIdx.x * NB + threadIdx.x;
    real hmin = real(3.0e38), hmax = 0, mmin = real(3.0e38), mmax = 0;
    if (gidx < n) {
        int a = 0;
        while (a + 1 < A.na && gidx >= A.base[a + 1]) ++a;
        const long long i = gidx - A.base[a];
        const PackSrc s = A.a[a];
        const real h = s.h[i];
        const real rho = s.rho ? s.rho[i] : pc.rho0;
        const real p = s.p ? s.p[i] : eos_pressure(rho, pc.rho0, pc.B, pc.gamma, pc.gamma_is_7);
        S.posh[gidx] = make_real4(s.x[i], s.y[i], s.z ? s.z[i] : real(0), h);
        S.velm[gidx] = make_real4(s.u ? s.u[i] : real(0), s.v ? s.v[i] : real(0), s.w ? s.w[i] : real(0), s.m ? s.m[i] : real(0));
        S.rp[gidx] = make_real2(rho, p / (rho * rho));
        S.meta[gidx] = ((uint32_t)a << SPH_META_IDX_BITS) | (uint32_t)i;
        S.acc[gidx] = make_real4(s.ax ? s.ax[i] : real(0), s.ay ? s.ay[i] : real(0), s.az ? s.az[i] : real(0),
                                 s.arho ? s.arho[i] : real(0));
        hmin = hmax = h;
        mmin = mmax = fabs(s.m ? s.m[i] : real(0));
    }
    real_bits bhmin = real_as_bits(hmin), bhmax = real_as_bits(hmax), bmmin = real_as_bits(mmin), bmmax = real_as_bits(mmax);
    for (int o = 16; o > 0; o >>= 1) {
        bhmin = min(bhmin, shfl_xor_bits(bhmin, o)); bhmax = max(bhmax, shfl_xor_bits(bhmax, o));
        bmmin = min(bmmin, shfl_xor_bits(bmmin, o)); bmmax = max(bmmax, shfl_xor_bits(bmmax, o));
    }
    if ((threadIdx.x & 31) == 0 && bhmax > 0) {        // positive reals order like their bit patterns
        atomicMin(&hminmax[0], bhmin);
        atomicMax(&hminmax[1], bhmax);
        atomicMin(&hminmax[2], bmmin);                 // |m|: uniform mass is detected for the UM / VU state layouts
        atomicMax(&hminmax[3], bmmax);
    }
}

__global__ void __launch_bounds__(NB)
k_key_hist(GridDesc g, SortedState S, int n, uint32_t* __restrict__ key, uint32_t* __restrict__ rank,
           uint32_t* __restrict__ cell_count, unsigned long long* __restrict__ counters) {
    const int i = blockIdx.x * NB + threadIdx.x;
    if (i >= n) return;
    bool oob;
    const float4 p = to_float4(S.posh[i]);                            // posh.w is still h here (k_pack; the layouts change at the sort)
    const uint32_t cell = cell_of(g, p, level_of_h(g, p.w), oob);
    const uint32_t k = cell * (uint32_t)g.na + (S.meta[i] >> SPH_META_IDX_BITS);
    SPH_DBG_ASSERT(cell < g.cells_total, g);
    key[i] = k;
    rank[i] = atomicAdd(&cell_count[k], 1u);
    if (oob) atomicAdd(&counters[CNT_OUT_OF_DOMAIN], 1ull);
}

// ------------------------------------------------------------------------------------------------
// a8 + a1 fused: [finish step n: u += dt/2 a] + [start step n+1: u += dt/2 a; x += dt u; wrap] + cell key +
// histogram.  eqs. 12-14 (L148-152); update_domain() periodic wrap (L443).  Continuity mode steps rho the same
// way on EVERY array (the tank particles too, L142) and re-evaluates the EOS (group 1 of Listing 3).
// ------------------------------------------------------------------------------------------------
struct UpdateArgs {
    real dt_half, dt; int kick2, kick1, move, continuity, rekey, w_rho, w_prr, euler, zero_cnt;
    int fixed[SPH_MAX_ARRAYS];
};

__global__ void __launch_bounds__(NB)
k_update(GridDesc g, PairConsts pc, SortedState S, int n, UpdateArgs U,
         uint32_t* __restrict__ key, uint32_t* __restrict__ rank, uint32_t* __restrict__ cell_count,
         unsigned long long* __restrict__ counters) {
    const int i = blockIdx.x * NB + threadIdx.x;
    // inside sph_pc_step this launch precedes the search and the pair passes of the step: it clears their counters
    // (no separate memset node per step)
    if (U.zero_cnt && i < CNT_COUNT - CNT_PAIRS_DENSITY) counters[CNT_PAIRS_DENSITY + i] = 0ull;
    if (i >= n) return;
    real4 pos = S.posh[i];
    const uint32_t meta = S.meta[i];
    const uint32_t aid = meta >> SPH_META_IDX_BITS;
    const real4 a = S.acc[i];
    if (!U.fixed[aid]) {
        real4 vel = S.velm[i];
        if (U.kick2) {                                                  // eq.14
            vel.x = rfma(U.dt_half, a.x, vel.x); vel.y = rfma(U.dt_half, a.y, vel.y);
            if (g.dim == 3) vel.z = rfma(U.dt_half, a.z, vel.z);
        }
        if (U.euler && U.move) {                                        // forward Euler: x^{n+1} = x^n + dt u^n (old u)
            pos.x = rfma(U.dt, vel.x, pos.x); pos.y = rfma(U.dt, vel.y, pos.y);
            if (g.dim == 3) pos.z = rfma(U.dt, vel.z, pos.z);
        }
        if (U.kick1) {
            vel.x = rfma(U.dt_half, a.x, vel.x); vel.y = rfma(U.dt_half, a.y, vel.y);   // eq.12
            if (g.dim == 3) vel.z = rfma(U.dt_half, a.z, vel.z);
            if (U.move) {                                                // eq.13 + periodic wrap
                if (!U.euler) {
                    pos.x = rfma(U.dt, vel.x, pos.x); pos.y = rfma(U.dt, vel.y, pos.y);
                    if (g.dim == 3) pos.z = rfma(U.dt, vel.z, pos.z);
                }
                if (g.per[0]) { if (pos.x >= g.hir[0]) pos.x -= g.Lr[0]; else if (pos.x < g.lor[0]) pos.x += g.Lr[0]; }
                if (g.per[1]) { if (pos.y >= g.hir[1]) pos.y -= g.Lr[1]; else if (pos.y < g.lor[1]) pos.y += g.Lr[1]; }
                if (g.dim == 3 && g.per[2]) { if (pos.z >= g.hir[2]) pos.z -= g.Lr[2]; else if (pos.z < g.lor[2]) pos.z += g.Lr[2]; }
                S.posh[i] = pos;
            }
        }
        S.velm[i] = vel;
    }
    if (U.continuity) {
        real rho = S.rp[i].x;
        if (U.kick2) rho = rfma(U.dt_half, a.w, rho);
        if (U.kick1) rho = rfma(U.dt_half, a.w, rho);
        const real p = eos_pressure(rho, pc.rho0, pc.B, pc.gamma, pc.gamma_is_7);
        S.rp[i] = make_real2(rho, p / (rho * rho));
        if (U.w_rho) S.velm[i].w = rho;         // constant h: velm.w of the sorted state carries rho (SortedState)
        if (U.w_prr) S.posh[i].w = p / (rho * rho);   // ... and, with uniform mass, posh.w carries p/rho^2
    }
    if (U.rekey) {
        bool oob;
        const float4 posf = to_float4(pos);
        const uint32_t cell = cell_of(g, posf, g.nlev > 1 ? level_of_h(g, posf.w) : 0, oob);   // several levels only when h varies: posh.w = h
        const uint32_t k = cell * (uint32_t)g.na + aid;
        SPH_DBG_ASSERT(cell < g.cells_total, g);
        key[i] = k;
        rank[i] = atomicAdd(&cell_count[k], 1u);
        if (oob) atomicAdd(&counters[CNT_OUT_OF_DOMAIN], 1ull);
    }
}

// ------------------------------------------------------------------------------------------------
// exclusive scan of n uint32 (out has n+1 entries; out[n] = total), one launch.
// ------------------------------------------------------------------------------------------------
#define SCAN_T 512
#ifndef SCAN_ITEMS
#define SCAN_ITEMS 8                 // two 16-byte vectors per thread (4: k_scan 367 us on C5's 51 M keys, 8: 243 us)
#endif
#define SCAN_TILE (SCAN_T * SCAN_ITEMS)

__device__ __forceinline__ uint32_t block_exclusive_scan(uint32_t v, uint32_t* total) {
    __shared__ uint32_t warp_sums[SCAN_T / 32];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    uint32_t inc = v;
    for (int o = 1; o < 32; o <<= 1) { uint32_t t = __shfl_up_sync(SPH_FULL_MASK, inc, o); if (lane >= o) inc += t; }
    if (lane == 31) warp_sums[w] = inc;
    __syncthreads();
    if (w == 0) {
        uint32_t s = lane < SCAN_T / 32 ? warp_sums[lane] : 0u, si = s;
        for (int o = 1; o < 32; o <<= 1) { uint32_t t = __shfl_up_sync(SPH_FULL_MASK, si, o); if (lane >= o) si += t; }
        if (lane < SCAN_T / 32) warp_sums[lane] = si - s;
        if (lane == 31 && total) *total = si;
    }
    __syncthreads();
    const uint32_t r = warp_sums[w] + inc - v;
    __syncthreads();
    return r;
}

// Single-pass scan with decoupled look-back: tile t publishes its aggregate, then warp 0 sums the aggregates of
// its predecessors, 32 at a time, back to the nearest tile whose inclusive prefix is already known.  Tiles take
// their number from a ticket, so every predecessor of a running tile is running or done (no deadlock).  A state
// word is {epoch-tagged flag, value}; the epoch (a device word) changes with every scan, so the table is never cleared.
__global__ void __launch_bounds__(SCAN_T)
k_scan(uint32_t* __restrict__ in, long long n, uint32_t* __restrict__ out, int nb,
       unsigned long long* __restrict__ state, uint32_t* __restrict__ ticket, int zero_in) {
    __shared__ uint32_t s_tile, s_total, s_prefix, s_epoch;
    if (threadIdx.x == 0) {
        s_epoch = *(volatile uint32_t*)(ticket + 1) + 1u;      // the epoch lives on the device (ticket[1]) so that a captured
        __threadfence_block();                                 // launch can be replayed; read BEFORE the ticket is taken: the
        s_tile = atomicAdd(ticket, 1u);                        // last tile bumps it only after every tile holds a ticket
    }
    __syncthreads();
    const uint32_t tile = s_tile, epoch = s_epoch;
    const long long i0 = (long long)tile * SCAN_TILE + (long long)threadIdx.x * SCAN_ITEMS;
    uint32_t v[SCAN_ITEMS], s = 0;
    const bool full = i0 + SCAN_ITEMS <= n;                              // 16-byte vector path (i0 % 4 == 0)
    if (full) {
#pragma unroll
        for (int k = 0; k < SCAN_ITEMS; k += 4) {
            const uint4 q = *reinterpret_cast<const uint4*>(in + i0 + k);
            v[k] = q.x; v[k + 1] = q.y; v[k + 2] = q.z; v[k + 3] = q.w; s += q.x + q.y + q.z + q.w;
            if (zero_in) *reinterpret_cast<uint4*>(in + i0 + k) = make_uint4(0u, 0u, 0u, 0u);   // the histogram is consumed: leave it cleared for the next step
        }
    } else {
#pragma unroll
        for (int k = 0; k < SCAN_ITEMS; ++k) { v[k] = (i0 + k < n) ? in[i0 + k] : 0u; s += v[k]; }
        if (zero_in) {
#pragma unroll
            for (int k = 0; k < SCAN_ITEMS; ++k) if (i0 + k < n) in[i0 + k] = 0u;
        }
    }
    uint32_t ex = block_exclusive_scan(s, &s_total);
    __syncthreads();
    const uint32_t total = s_total;
    const uint32_t F_AGG = 2u * epoch + 1u, F_INC = 2u * epoch + 2u;
    volatile unsigned long long* vs = state;
    if (threadIdx.x < 32) {
        const int lane = threadIdx.x;
        uint32_t prefix = 0u;
        if (tile > 0) {
            if (lane == 0) vs[tile] = ((unsigned long long)F_AGG << 32) | total;
            long long p = (long long)tile - 1;                    // look back over tiles p, p-1, ... (lane = distance)
            for (;;) {
                const long long q = p - lane;
                unsigned long long w = 0ull; uint32_t f = F_INC;   // tiles before 0 count as "inclusive, 0"
                if (q >= 0) { do { w = vs[q]; f = (uint32_t)(w >> 32); } while (f != F_AGG && f != F_INC); }
                const unsigned inc = __ballot_sync(SPH_FULL_MASK, f == F_INC);
                const int stop = inc ? __ffs(inc) - 1 : 32;        // nearest tile with a known inclusive prefix
                uint32_t add = (lane <= stop && q >= 0) ? (uint32_t)w : 0u;
                for (int o = 16; o > 0; o >>= 1) add += __shfl_xor_sync(SPH_FULL_MASK, add, o);
                prefix += add;
                if (inc) break;
                p -= 32;
            }
        }
        if (lane == 0) {
            vs[tile] = ((unsigned long long)F_INC << 32) | (prefix + total);
            s_prefix = prefix;
            if ((int)tile == nb - 1) {                                  // last tile: grand total, ticket reset, next epoch
                out[n] = prefix + total; ticket[1] = epoch >= 0x3ffffff0u ? 0u : epoch; ticket[0] = 0u;
            }
        }
    }
    __syncthreads();
    ex += s_prefix;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) { const uint32_t e = ex; ex += v[k]; v[k] = e; }
    if (full) {
#pragma unroll
        for (int k = 0; k < SCAN_ITEMS; k += 4) *reinterpret_cast<uint4*>(out + i0 + k) = make_uint4(v[k], v[k + 1], v[k + 2], v[k + 3]);
    }
    else {
#pragma unroll
        for (int k = 0; k < SCAN_ITEMS; ++k) if (i0 + k < n) out[i0 + k] = v[k];
    }
}

// Large tables (>= SCAN_TWO_LEVEL_TILES tiles): reduce -> scan of the tile sums -> scan with the known tile prefix.
// It reads the table twice (16 B per key with the clearing instead of 12) but has no look-back: in the single-pass
// kernel a tile holds its SM slot for ~11 us, 7 of them waiting for the flags of its predecessors (ncu: `barrier`
// stalls; a microbenchmark of the same kernel without the look-back runs at 4.9 TB/s, with it at 2.0), whatever the
// width of the look-back window.  Small tables keep the single launch.
#ifndef SCAN_TWO_LEVEL_TILES
#define SCAN_TWO_LEVEL_TILES 1024
#endif
__global__ void __launch_bounds__(SCAN_T)
k_scan_reduce(const uint32_t* __restrict__ in, long long n, uint32_t* __restrict__ tile_sum) {
    __shared__ uint32_t s_w[SCAN_T / 32];
    const long long i0 = (long long)blockIdx.x * SCAN_TILE + (long long)threadIdx.x * SCAN_ITEMS;
    uint32_t s = 0;
    if (i0 + SCAN_ITEMS <= n) {
#pragma unroll
        for (int k = 0; k < SCAN_ITEMS; k += 4) { const uint4 q = *reinterpret_cast<const uint4*>(in + i0 + k); s += q.x + q.y + q.z + q.w; }
    } else {
#pragma unroll
        for (int k = 0; k < SCAN_ITEMS; ++k) s += (i0 + k < n) ? in[i0 + k] : 0u;
    }
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(SPH_FULL_MASK, s, o);
    if ((threadIdx.x & 31) == 0) s_w[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x < 32) {
        uint32_t t = threadIdx.x < SCAN_T / 32 ? s_w[threadIdx.x] : 0u;
        for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(SPH_FULL_MASK, t, o);
        if (threadIdx.x == 0) tile_sum[blockIdx.x] = t;
    }
}

// one block: tile_prefix[t] = sum of tile_sum[0..t), tile_prefix[nb] = total (nb <= 1024 * 64)
__global__ void __launch_bounds__(1024)
k_scan_tiles(const uint32_t* __restrict__ tile_sum, int nb, uint32_t* __restrict__ tile_prefix) {
    __shared__ uint32_t s_w[32];
    const int per = (nb + 1023) / 1024, lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int b = threadIdx.x * per, e = min(b + per, nb);
    uint32_t s = 0;
    for (int k = b; k < e; ++k) s += tile_sum[k];
    uint32_t inc = s;
    for (int o = 1; o < 32; o <<= 1) { const uint32_t t = __shfl_up_sync(SPH_FULL_MASK, inc, o); if (lane >= o) inc += t; }
    if (lane == 31) s_w[w] = inc;
    __syncthreads();
    if (w == 0) {
        const uint32_t v = s_w[lane]; uint32_t vi = v;
        for (int o = 1; o < 32; o <<= 1) { const uint32_t t = __shfl_up_sync(SPH_FULL_MASK, vi, o); if (lane >= o) vi += t; }
        s_w[lane] = vi - v;
        if (lane == 31) tile_prefix[nb] = vi;
    }
    __syncthreads();
    uint32_t run = s_w[w] + inc - s;
    for (int k = b; k < e; ++k) { tile_prefix[k] = run; run += tile_sum[k]; }
}

__global__ void __launch_bounds__(SCAN_T)
k_scan_apply(uint32_t* __restrict__ in, long long n, uint32_t* __restrict__ out, const uint32_t* __restrict__ tile_prefix, int nb, int zero_in) {
    __shared__ uint32_t s_total;
    const long long i0 = (long long)blockIdx.x * SCAN_TILE + (long long)threadIdx.x * SCAN_ITEMS;
    uint32_t v[SCAN_ITEMS], s = 0;
    const bool full = i0 + SCAN_ITEMS <= n;
    if (full) {
#pragma unroll
        for (int k = 0; k < SCAN_ITEMS; k += 4) {
            const uint4 q = *reinterpret_cast<const uint4*>(in + i0 + k);
            v[k] = q.x; v[k + 1] = q.y; v[k + 2] = q.z; v[k + 3] = q.w; s += q.x + q.y + q.z + q.w;
            if (zero_in) *reinterpret_cast<uint4*>(in + i0 + k) = make_uint4(0u, 0u, 0u, 0u);
        }
    } else {
#pragma unroll
        for (int k = 0; k < SCAN_ITEMS; ++k) { v[k] = (i0 + k < n) ? in[i0 + k] : 0u; s += v[k]; }
        if (zero_in) {
#pragma unroll
            for (int k = 0; k < SCAN_ITEMS; ++k) if (i0 + k < n) in[i0 + k] = 0u;
        }
    }
    uint32_t ex = block_exclusive_scan(s, &s_total) + __ldg(tile_prefix + blockIdx.x);
    if ((int)blockIdx.x == nb - 1 && threadIdx.x == 0) out[n] = __ldg(tile_prefix + nb);
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) { const uint32_t e = ex; ex += v[k]; v[k] = e; }
    if (full) {
#pragma unroll
        for (int k = 0; k < SCAN_ITEMS; k += 4) *reinterpret_cast<uint4*>(out + i0 + k) = make_uint4(v[k], v[k + 1], v[k + 2], v[k + 3]);
    } else {
#pragma unroll
        for (int k = 0; k < SCAN_ITEMS; ++k) if (i0 + k < n) out[i0 + k] = v[k];
    }
}

static int scan_exclusive(sph_ctx* c, uint32_t* in, uint32_t* out, long long n, bool zero_in) {
    const int nb = (int)((n + SCAN_TILE - 1) / SCAN_TILE);
    if (nb == 0) { SPH_CUDA_OK(c, cudaMemsetAsync(out, 0, sizeof(uint32_t), c->stream)); return SPH_OK; }
    if (nb >= SCAN_TWO_LEVEL_TILES && nb <= c->scan_tiles_cap) {
        uint32_t* tile_sum = c->scan_tiles; uint32_t* tile_prefix = c->scan_tiles + c->scan_tiles_cap + 1;
        SPH_LAUNCH(c, SPH_K_SCAN_REDUCE, k_scan_reduce, nb, SCAN_T, 0, in, n, tile_sum);
        SPH_LAUNCH(c, SPH_K_SCAN_TILES, k_scan_tiles, 1, 1024, 0, tile_sum, nb, tile_prefix);
        SPH_LAUNCH(c, SPH_K_SCAN, k_scan_apply, nb, SCAN_T, 0, in, n, out, tile_prefix, nb, zero_in ? 1 : 0);
        return SPH_OK;
    }
    SPH_LAUNCH(c, SPH_K_SCAN, k_scan, nb, SCAN_T, 0, in, n, out, nb, c->scan_state, c->scan_ticket, zero_in ? 1 : 0);
    return SPH_OK;
}

// a3: gather every persistent property into cell order (double buffer A -> B).
__global__ void __launch_bounds__(NB)
k_scatter(GridDesc g, SortedState A, SortedState B, int n, int na, int with_acc, int w_mass, const uint32_t* __restrict__ key,
          const uint32_t* __restrict__ rank, const uint32_t* __restrict__ cell_start, uint32_t* __restrict__ nl_head) {
    const int i = blockIdx.x * NB + threadIdx.x;
    if (i >= n) return;
    const uint32_t k = key[i];
    const uint32_t d = cell_start[k] + rank[i];
    SPH_DBG_ASSERT(k / (uint32_t)na < g.cells_total && d < (uint32_t)n, g);
    real4 p = A.posh[i];
    real4 v = A.velm[i];
    const real2 r = A.rp[i];
    // first sort after the pack (SortedState).  constant h: velm.w <- rho; posh.w <- m, or <- p/rho^2 when the mass is uniform
    if (w_mass == 3) v.w = r.x;                                      // VU layout (variable h): velm.w <- rho, posh.w stays h
    else if (w_mass) { p.w = w_mass == 2 ? r.y : v.w; v.w = r.x; }
    B.posh[d] = p;
    B.velm[d] = v;
    B.rp[d] = r;
    B.meta[d] = A.meta[i];
    B.cell[d] = k / (uint32_t)na;
    if (nl_head && (d & 31u) == 0u) nl_head[d >> 5] = 0u;          // the records of the old order are void: clear the heads for the next search
    if (with_acc) B.acc[d] = A.acc[i];
}

int nnps_key_hist(sph_ctx* c) {
    const int n = (int)c->n_total;
    // cell_count is clear here: sph_nnps_build clears it after sizing the grid, every scan leaves it cleared
    if (n) SPH_LAUNCH(c, SPH_K_KEY, k_key_hist, (n + NB - 1) / NB, NB, 0, c->grid, c->S[c->cur], n, c->key, c->rank,
                      c->cell_count, c->counters);
    return SPH_OK;
}

int nnps_update_key_hist(sph_ctx* c, real dt, bool kick2, bool kick1_drift, bool continuity, bool rekey) {
    const bool kick_only = kick2 && !kick1_drift;
    const int n = (int)c->n_total;
    UpdateArgs U;
    U.euler = c->prm.integrator == SPH_INTEGRATOR_EULER ? 1 : 0;
    U.dt_half = U.euler ? dt : real(0.5) * dt;              // Euler: the one kick per step is a full dt
    U.dt = dt; U.kick2 = kick2; U.kick1 = kick1_drift; U.move = c->prm.move;
    U.continuity = continuity; U.rekey = rekey; U.zero_cnt = rekey ? 1 : 0; U.w_rho = (!c->variable_h || c->pc.varh_um) ? 1 : 0; U.w_prr = (!c->variable_h && c->pc.uniform_m) ? 1 : 0;
    for (int a = 0; a < SPH_MAX_ARRAYS; ++a) U.fixed[a] = a < c->na ? c->fixed[a] : 1;
    if (n) SPH_LAUNCH(c, (kick_only ? SPH_K_UPDATE_KICK : SPH_K_UPDATE), k_update, (n + NB - 1) / NB, NB, 0, c->grid, c->pc, c->S[c->cur], n, U, c->key, c->rank,
                      c->cell_count, c->counters);
    if (n && rekey) c->counters_fresh = true;
    return SPH_OK;
}

int nnps_sort_from_keys(sph_ctx* c, bool with_acc) {
    const int n = (int)c->n_total;
    int rc = scan_exclusive(c, c->cell_count, c->cell_start, c->n_keys, true);   // leaves cell_count cleared
    if (rc) return rc;
    if (n) SPH_LAUNCH(c, SPH_K_SCATTER, k_scatter, (n + NB - 1) / NB, NB, 0, c->grid, c->S[c->cur], c->S[c->cur ^ 1], n, c->na,
                      with_acc ? 1 : 0, !with_acc ? 0 : (c->variable_h ? (c->pc.varh_um ? 3 : 0) : (c->pc.uniform_m ? 2 : 1)), c->key, c->rank, c->cell_start, c->nl.head);
    c->heads_fresh = n > 0 && c->nl.head != nullptr;
    c->cur ^= 1;
    c->nl_valid = false;                 // recorded neighbour rows index the previous sorted order
    c->inv_valid = false;
    return SPH_OK;
}

// ------------------------------------------------------------------------------------------------
// caller-order outputs
// ------------------------------------------------------------------------------------------------
// inv[base(array) + original index] = sorted index: the caller-order outputs then WRITE coalesced (one thread per
// caller-order particle) instead of scattering 4-byte words (8x write amplification at 32-byte sectors)
__global__ void __launch_bounds__(NB)
k_inverse(SortedState S, int n, PackArgs A, uint32_t* __restrict__ inv) {
    const int i = blockIdx.x * NB + threadIdx.x;
    if (i >= n) return;
    const uint32_t meta = S.meta[i];
    inv[A.base[meta >> SPH_META_IDX_BITS] + (long long)(meta & SPH_META_IDX_MASK)] = (uint32_t)i;
}

__global__ void __launch_bounds__(NB)
k_gather_out(SortedState S, int n_array, const uint32_t* __restrict__ inv, OutPtrs O) {
    const int o = blockIdx.x * NB + threadIdx.x;
    if (o >= n_array) return;
    const uint32_t i = inv[o];
    if (O.x || O.y || O.z) { const real4 p = S.posh[i]; if (O.x) O.x[o] = p.x; if (O.y) O.y[o] = p.y; if (O.z) O.z[o] = p.z; }
    if (O.u || O.v || O.w) { const real4 v = S.velm[i]; if (O.u) O.u[o] = v.x; if (O.v) O.v[o] = v.y; if (O.w) O.w[o] = v.z; }
    if (O.rho || O.p) { const real2 r = S.rp[i]; if (O.rho) O.rho[o] = r.x; if (O.p) O.p[o] = r.y * r.x * r.x; }
    if (O.ax || O.ay || O.az || O.arho) {
        const real4 a = S.acc[i];
        if (O.ax) O.ax[o] = a.x; if (O.ay) O.ay[o] = a.y; if (O.az) O.az[o] = a.z; if (O.arho) O.arho[o] = a.w;
    }
}

int nnps_gather_out(sph_ctx* c, int array, const OutPtrs& O) {
    const int n = (int)c->n_total;
    if (n == 0 || c->n[array] == 0) return SPH_OK;
    if (!c->inv_valid) {                       // once per sorted order (rank is idle between sorts)
        PackArgs A; memset(&A, 0, sizeof(A));
        A.na = c->na;
        for (int a = 0; a <= c->na; ++a) A.base[a] = c->base[a];
        SPH_LAUNCH(c, SPH_K_OUTPUT, k_inverse, (n + NB - 1) / NB, NB, 0, c->S[c->cur], n, A, c->rank);
        c->inv_valid = true;
    }
    const int na_ = (int)c->n[array];
    SPH_LAUNCH(c, SPH_K_OUTPUT, k_gather_out, (na_ + NB - 1) / NB, NB, 0, c->S[c->cur], na_, c->rank + c->base[array], O);
    return SPH_OK;
}

// ------------------------------------------------------------------------------------------------
// neighbour-list export (verification): the same warp-tile walker and predicate code as the pair kernels.
// ------------------------------------------------------------------------------------------------
struct NbSrc { real4 pj; uint32_t meta; };

template <int DIM, bool VARH, bool FILL>
__global__ void __launch_bounds__(TILE_BLOCK)
k_neighbors_tile(GridDesc g, PairConsts pc, SortedState S, const uint32_t* __restrict__ cell_start, int n,
                 uint32_t dest, uint32_t src, uint32_t* __restrict__ counts, const uint32_t* __restrict__ offsets,
                 int32_t* __restrict__ indices) {
    typedef TileWarpSmemT<TILE_MMAX_OF(VARH)> WS;
    __shared__ WS smem[TILE_WARPS];
    WS& ws = smem[threadIdx.x >> 5];
    const int i = blockIdx.x * TILE_BLOCK + threadIdx.x;
    const bool in = i < n;
    uint32_t meta = 0, ci = 0; real4 pi = make_real4(0, 0, 0, 1);
    if (in) { meta = S.meta[i]; ci = S.cell[i]; pi = S.posh[i]; }
    const bool active = in && (meta >> SPH_META_IDX_BITS) == dest;
    if (!__any_sync(SPH_FULL_MASK, active)) return;
    const uint32_t o = meta & SPH_META_IDX_MASK;
    const real hi = VARH ? pi.w : pc.h_const, kh = sizeof(real) == 8 ? pc.ksup : pc.kh;
    const real cut2c = pair_cut2(kh, pc.h_const, pc.h_const);
    uint32_t cnt = 0;
    int32_t* out = FILL ? indices + (active ? offsets[o] : 0u) : nullptr;
    auto load = [&](uint32_t j) { NbSrc s; s.pj = ldg_r(S.posh + j); s.meta = __ldg(S.meta + j); return s; };
    auto compute = [&](const NbSrc& s, bool has, uint32_t code, auto per) {
        real dx = rsub(pi.x, s.pj.x), dy = rsub(pi.y, s.pj.y), dz = DIM == 3 ? rsub(pi.z, s.pj.z) : real(0);
        if (decltype(per)::value) {
            dx = rsub(dx, img_shift(code, 0, g.Lr[0])); dy = rsub(dy, img_shift(code, 1, g.Lr[1]));
            if (DIM == 3) dz = rsub(dz, img_shift(code, 2, g.Lr[2]));
        }
        has = has && pair_r2(dx, dy, dz) < (VARH ? pair_cut2(kh, hi, s.pj.w) : cut2c);     // the exact predicate R7
        if (!has || (s.meta >> SPH_META_IDX_BITS) != src) return;
        if (FILL) out[cnt] = (int32_t)(s.meta & SPH_META_IDX_MASK);
        ++cnt;
    };
    TileState st; st.reset(); st.tests = 0;
    const uint32_t idle = in ? (uint32_t)i : 0u;
    tile_walk<DIM, VARH>(g, pc, S.posh, cell_start, active, in, to_float4(pi), ci, ws, st, [&]() {
        if (st.shifted) tile_drain<NbSrc, 2, true>(ws, st.nz, idle, load, compute);
        else            tile_drain<NbSrc, 2, false>(ws, st.nz, idle, load, compute);
        st.reset(); });
    if (!active) return;
    if (!FILL) counts[o] = cnt;
    else {                                              // rows ascending (insertion sort; rows are short)
        const int m = (int)cnt;
        for (int a = 1; a < m; ++a) { int32_t v = out[a]; int b = a - 1; while (b >= 0 && out[b] > v) { out[b + 1] = out[b]; --b; } out[b + 1] = v; }
    }
}

__global__ void k_widen(const uint32_t* __restrict__ in, int64_t* __restrict__ out, long long n) {
    const long long i = (long long)blockIdx.x * NB + threadIdx.x;
    if (i < n) out[i] = (int64_t)in[i];
}

int nnps_export_neighbors(sph_ctx* c, int dest, int src, int64_t* offsets, int32_t* indices, int64_t cap,
                          int64_t* total, int mem) {
    const int n = (int)c->n_total;
    const long long nd = c->n[dest];
    uint32_t* counts = c->key;            // scratch: key/rank are dead between sorts
    uint32_t* off32 = c->rank;
    c->inv_valid = false;                 // (rank also holds the inverse permutation of the caller-order outputs)
    SPH_CUDA_OK(c, cudaMemsetAsync(counts, 0, (size_t)(nd + 1) * sizeof(uint32_t), c->stream));
    SortedState& S = c->S[c->cur];
    const int tgrid = (n + TILE_BLOCK - 1) / TILE_BLOCK;
#define LN(FILL, IDX) do { \
    if (c->grid.dim == 2) { if (c->variable_h) SPH_LAUNCH(c, SPH_K_NEIGHBORS, (k_neighbors_tile<2, true, FILL>), tgrid, TILE_BLOCK, 0, c->grid, c->pc, S, c->cell_start, n, (uint32_t)dest, (uint32_t)src, counts, off32, IDX); \
                            else SPH_LAUNCH(c, SPH_K_NEIGHBORS, (k_neighbors_tile<2, false, FILL>), tgrid, TILE_BLOCK, 0, c->grid, c->pc, S, c->cell_start, n, (uint32_t)dest, (uint32_t)src, counts, off32, IDX); } \
    else                  { if (c->variable_h) SPH_LAUNCH(c, SPH_K_NEIGHBORS, (k_neighbors_tile<3, true, FILL>), tgrid, TILE_BLOCK, 0, c->grid, c->pc, S, c->cell_start, n, (uint32_t)dest, (uint32_t)src, counts, off32, IDX); \
                            else SPH_LAUNCH(c, SPH_K_NEIGHBORS, (k_neighbors_tile<3, false, FILL>), tgrid, TILE_BLOCK, 0, c->grid, c->pc, S, c->cell_start, n, (uint32_t)dest, (uint32_t)src, counts, off32, IDX); } } while (0)
    if (n) LN(false, (int32_t*)nullptr);
    int rc = scan_exclusive(c, counts, off32, nd, false);
    if (rc) return rc;
    uint32_t tot32 = 0;
    SPH_CUDA_OK(c, cudaMemcpyAsync(&tot32, off32 + nd, sizeof(uint32_t), cudaMemcpyDeviceToHost, c->stream));
    SPH_CUDA_OK(c, cudaStreamSynchronize(c->stream));
    *total = (int64_t)tot32;
    int64_t* d_off = offsets; int32_t* d_idx = indices;
    if (mem == SPH_MEM_HOST) {            // verification-only path: temporary device buffers
        SPH_CUDA_OK(c, cudaMalloc(&d_off, (size_t)(nd + 1) * sizeof(int64_t)));
        if (indices && cap >= *total && *total > 0) SPH_CUDA_OK(c, cudaMalloc(&d_idx, (size_t)(*total) * sizeof(int32_t)));
    }
    SPH_LAUNCH(c, SPH_K_NEIGHBORS, k_widen, (int)((nd + 1 + NB - 1) / NB), NB, 0, off32, d_off, nd + 1);
    const bool fill = indices && cap >= *total && *total > 0;
    if (fill && n) LN(true, d_idx);
#undef LN
    if (mem == SPH_MEM_HOST) {
        SPH_CUDA_OK(c, cudaMemcpyAsync(offsets, d_off, (size_t)(nd + 1) * sizeof(int64_t), cudaMemcpyDeviceToHost, c->stream));
        if (fill) SPH_CUDA_OK(c, cudaMemcpyAsync(indices, d_idx, (size_t)(*total) * sizeof(int32_t), cudaMemcpyDeviceToHost, c->stream));
        SPH_CUDA_OK(c, cudaStreamSynchronize(c->stream));
        cudaFree(d_off); if (fill) cudaFree(d_idx);
    } else SPH_CUDA_OK(c, cudaStreamSynchronize(c->stream));
    return SPH_OK;
}

// ------------------------------------------------------------------------------------------------
// build entry used by sph_nnps_build: pack -> (host sizes the grid from h_max) -> key/hist -> sort
// ------------------------------------------------------------------------------------------------
int nnps_pack(sph_ctx* c, const PackArgs& A) {
    const int n = (int)c->n_total;
    const real big = real(3.0e38);
    real_bits init[4] = { 0, 0, 0, 0 };
    memcpy(&init[0], &big, sizeof(real)); memcpy(&init[2], &big, sizeof(real));
    SPH_CUDA_OK(c, cudaMemcpyAsync(c->hminmax, init, sizeof(init), cudaMemcpyHostToDevice, c->stream));
    if (n) SPH_LAUNCH(c, SPH_K_PACK, k_pack, (n + NB - 1) / NB, NB, 0, A, c->S[c->cur], n, c->pc, (real_bits*)c->hminmax);
    return SPH_OK;
}

// ------------------------------------------------------------------------------------------------
// Diagnostic: size of the candidate set of the PAPER's cell-list search (L158: "3^d neighbouring boxes" of a
// uniform grid with cells >= k h_max): sum over particles of the population of the 3^d coarse cells around them.
// It is the algorithmic work unit of the searching passes in the roofline report.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void coarse_coords(const GridDesc& g, float4 p, int (&c)[3], int (&nc)[3]) {
    const LevelDesc& Lv = g.lev[g.nlev - 1];
    nc[0] = Lv.nc[0] / Lv.xsub; nc[1] = Lv.nc[1]; nc[2] = Lv.nc[2];
    c[0] = cell_coord(p.x, g.lo[0], Lv.inv_cell[0], Lv.nc[0]) / Lv.xsub;
    c[1] = cell_coord(p.y, g.lo[1], Lv.inv_cell[1], Lv.nc[1]);
    c[2] = g.dim == 3 ? cell_coord(p.z, g.lo[2], Lv.inv_cell[2], Lv.nc[2]) : 0;
}
__global__ void __launch_bounds__(NB)
k_coarse_hist(GridDesc g, SortedState S, int n, uint32_t* __restrict__ cnt) {
    const int i = blockIdx.x * NB + threadIdx.x;
    if (i >= n) return;
    int c[3], nc[3];
    coarse_coords(g, to_float4(S.posh[i]), c, nc);
    atomicAdd(&cnt[(c[2] * nc[1] + c[1]) * nc[0] + c[0]], 1u);
}
__global__ void __launch_bounds__(NB)
k_coarse_sum(GridDesc g, SortedState S, int n, const uint32_t* __restrict__ cnt, unsigned long long* __restrict__ out) {
    const int i = blockIdx.x * NB + threadIdx.x;
    unsigned long long sum = 0ull;
    if (i < n) {
        int c[3], nc[3];
        coarse_coords(g, to_float4(S.posh[i]), c, nc);
        for (int dz = (g.dim == 3 ? -1 : 0); dz <= (g.dim == 3 ? 1 : 0); ++dz)
            for (int dy = -1; dy <= 1; ++dy)
                for (int dx = -1; dx <= 1; ++dx) {
                    int q[3] = { c[0] + dx, c[1] + dy, c[2] + dz }; bool ok = true;
                    for (int a = 0; a < 3; ++a) {
                        if (q[a] < 0) { if (g.per[a]) q[a] += nc[a]; else ok = false; }
                        else if (q[a] >= nc[a]) { if (g.per[a]) q[a] -= nc[a]; else ok = false; }
                    }
                    if (ok) sum += cnt[(q[2] * nc[1] + q[1]) * nc[0] + q[0]];
                }
    }
    sum = warp_sum_u64(sum);
    if ((threadIdx.x & 31) == 0 && sum) atomicAdd(out, sum);
}

int nnps_stencil_candidates(sph_ctx* c, int64_t* out) {
    const int n = (int)c->n_total;
    *out = 0;
    if (n == 0) return SPH_OK;
    const LevelDesc& Lv = c->grid.lev[c->grid.nlev - 1];
    const size_t cells = (size_t)(Lv.nc[0] / Lv.xsub) * Lv.nc[1] * Lv.nc[2];
    unsigned long long* acc = (unsigned long long*)c->hminmax;                     // 16 bytes of scratch, idle between builds
    uint32_t* cnt = c->cell_count;                                                 // all zero between sorts; cleared again below
    SPH_CUDA_OK(c, cudaMemsetAsync(acc, 0, sizeof(unsigned long long), c->stream));
    SPH_LAUNCH(c, SPH_K_NEIGHBORS, k_coarse_hist, (n + NB - 1) / NB, NB, 0, c->grid, c->S[c->cur], n, cnt);
    SPH_LAUNCH(c, SPH_K_NEIGHBORS, k_coarse_sum, (n + NB - 1) / NB, NB, 0, c->grid, c->S[c->cur], n, cnt, acc);
    SPH_CUDA_OK(c, cudaMemsetAsync(cnt, 0, cells * sizeof(uint32_t), c->stream));
    unsigned long long h = 0;
    SPH_CUDA_OK(c, cudaMemcpyAsync(&h, acc, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    SPH_CUDA_OK(c, cudaStreamSynchronize(c->stream));
    *out = (int64_t)h;
    return SPH_OK;
}
