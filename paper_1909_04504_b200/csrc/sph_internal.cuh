// Internal declarations of the CUDA path (sm_100a).  Not part of the ABI; shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/sph.h"

// The real type of the particle state and of the field arithmetic: float (libsph_b200.so), or double when built with
// -DSPH_REAL_DOUBLE (libsph_b200_f64.so; north_star: "1e-12 for an fp64 build flag").  The neighbour SEARCH (cell
// coordinates, walker, tensor-core filter) always runs in float on float-rounded positions -- it is conservative by
// construction -- and the exact predicate and every field are evaluated in `real`.
#ifdef SPH_REAL_DOUBLE
typedef double real; typedef double2 real2; typedef double4 real4;
#define make_real2 make_double2
#define make_real4 make_double4
#else
typedef float real; typedef float2 real2; typedef float4 real4;
#define make_real2 make_float2
#define make_real4 make_float4
#endif

#define SPH_FULL_MASK 0xffffffffu
#define SPH_META_IDX_BITS 28u                    // meta = (array id << 28) | original index
#define SPH_META_IDX_MASK ((1u << SPH_META_IDX_BITS) - 1u)

// Cell grid (cells of size >= the support radius; L158-160, L171: one grid sized by h_max "becomes
// inefficient" when h varies).  Particles are binned by h into `nlev` LEVELS (geometric h classes; one level when h
// is constant); level l has its own uniform grid with cells >= k * hmax_l, all levels share ONE cell table and ONE
// sorted order (key = (level base + linear cell) * na + array, level-major).  In every level grid the y and z cells
// are >= the support radius of the level and every such cell is split into `xsub` sub-cells along x (x is the
// fastest key digit, so a stencil row is one contiguous run and an x-interval of it is a contiguous sub-run).
#define SPH_MAX_LEVELS 8
struct LevelDesc {
    int nc[3];                 // cells per axis (nc[2] = 1 in 2-D); nc[0] counts the x SUB-cells
    int xsub;                  // x sub-cells per support radius
    uint32_t base;             // first cell of this level in the shared cell table (in cells; times na = key)
    float inv_cell[3];         // 1 / cell size (x: sub-cell)
    float hmax;                // every particle binned into this level has h <= hmax
};
struct GridDesc {
    int dim;
    int na;                    // particle arrays merged into the grid: key = cell * na + array
    int nlev;                  // levels in use (1 when h is constant)
    int per[3];                // periodic per axis
    float lo[3];               // domain origin
    float L[3];                // (float)(hi - lo): the period used by the neighbour predicate (R7)
    real Lr[3];                // the same in the real type of the build (double build: hi - lo in double)
    real lor[3], hir[3];       // domain bounds in the real type (periodic wrap of eq.13)
    float hi[3];
    float uabs;                // 2^-23 * largest coordinate magnitude: absolute rounding unit of positions
    uint32_t n_sorted, cells_total;    // particles in the sorted order, cells of all level grids (bounds of the tables)
    unsigned long long* dbg;   // the context's device counters: -DSPH_DEBUG_ASSERT builds count failed bounds assertions there
    LevelDesc lev[SPH_MAX_LEVELS];
};
// Opt-in device-side bounds assertions (build with -DSPH_DEBUG_ASSERT; compute-sanitizer is closed on this pool): record-pool
// rows, cell-table and sorted-order indices, scan tiles.  A failure is counted and reported by the next [sync] call.
#define SPH_CNT_ASSERT 9
#ifdef SPH_DEBUG_ASSERT
#define SPH_DBG_ASSERT(cond, g) do { if (!(cond)) atomicAdd(&(g).dbg[SPH_CNT_ASSERT], 1ull); } while (0)
#else
#define SPH_DBG_ASSERT(cond, g) do { } while (0)
#endif

__host__ __device__ inline int level_of_h(const GridDesc& g, float h) {
    int l = 0;
    while (l + 1 < g.nlev && h > g.lev[l].hmax) ++l;
    return l;
}

// Candidate-mask records written by the search and replayed by the pair passes (sph_tile.cuh "mask records").  The
// pool is an array of ROWS of 32 words (one word per lane of the warp that owns the row); a warp appends contiguous
// BLOCKS: header row, shift-code row, one mask row per batch.
#define SPH_NL_NONE 0xffffffffu
struct NList {
    uint32_t* pool;            // pool_rows * 32 words
    uint32_t* head;            // per warp of the sorted order: first block (row index), 0 = none
    uint32_t* used;            // rows handed out so far (row 0 is reserved: allocation returns used + 1)
    uint32_t pool_rows;
};

// Per-launch constants of the pair loops.
struct PairConsts {
    real kh;                   // k/2: cut = kh * (h_i + h_j)
    real ksup;                 // k (the double build forms cut = k * (0.5 * (h_i + h_j)) like the oracle's double predicate)
    real sigma;                // kernel normalisation sigma_d
    real h_const;              // constant-h fast path: h, 1/h, sigma/h^d
    real hinv_const;
    real fac_const;
    real rho0, B, gamma;       // Tait EOS
    int   gamma_is_7;
    real visc;                 // -2 alpha c0   (Pi = visc * h vr / ((r2 + eps h^2)(rho_i + rho_j)))
    real eps;
    real m_const; int uniform_m;   // constant h and every particle of every array has the same mass: the UM layout
    int varh_um;               // variable h, uniform mass, gamma = 7 and p = EOS(rho): the VU layout (velm.w = rho, m = m_const)
    real nu4, eta;             // laminar viscosity eq.10: 4 nu (0 = term off) and its regulariser
    real g[3];
    uint32_t src_mask[SPH_MAX_ARRAYS];   // per DEST array: source-array bitmask; 0 = not a destination of this launch
    uint32_t all_mask;         // (1 << na) - 1
};

// Cell-sorted particle state (struct of float4 groups: one 16-B vector load per candidate test).
struct SortedState {
    real4* posh;               // x, y, z, h          | constant h (h_min == h_max; the kernels then take h from
    real4* velm;               // u, v, w, m          | PairConsts): after the sort velm = (u, v, w, RHO) and posh =
                               //                     | (x, y, z, M), so that the density pair loop gathers ONE 16-byte
                               //                     | word per neighbour and the momentum pair loop TWO (p/rho^2 is
                               //                     | recomputed from rho when p is the EOS of rho).  UM layout (all
                               //                     | masses equal too, PairConsts::uniform_m): posh = (x, y, z,
                               //                     | P/RHO^2) and the mass is the constant m_const: two gathers, no
                               //                     | recomputation.  VU layout (VARIABLE h, all masses equal, p is
                               //                     | the gamma = 7 EOS of rho; PairConsts::varh_um): posh = (x, y, z,
                               //                     | h), velm = (u, v, w, RHO), mass = m_const: the density loop gathers
                               //                     | one word per neighbour, the momentum loop two.
    real2* rp;                 // rho, p / rho^2   (p itself is returned as (p/rho^2) * rho^2)
    real4* acc;                // ax, ay, az, arho
    uint32_t* meta;            // (array << 28) | original index
    uint32_t* cell;            // linear cell id of the particle (x fastest)
};

// ---- device math ------------------------------------------------------------------------------
__device__ __forceinline__ float rcp_approx(float x)  { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float rsqrt_approx(float x){ float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

__device__ __forceinline__ float sqrt_approx(float x) { float y; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ double sqrt_approx(double x) { return sqrt(x); }
__device__ __forceinline__ double rcp_approx(double x)  { return 1.0 / x; }
__device__ __forceinline__ double rsqrt_approx(double x){ return 1.0 / sqrt(x); }
__device__ __forceinline__ float  rfma(float a, float b, float c)    { return fmaf(a, b, c); }
__device__ __forceinline__ double rfma(double a, double b, double c) { return fma(a, b, c); }
__device__ __forceinline__ float  rmax(float a, float b)   { return fmaxf(a, b); }
__device__ __forceinline__ double rmax(double a, double b) { return fmax(a, b); }
__device__ __forceinline__ float4 ldg_r(const float4* p) { return __ldg(p); }
__device__ __forceinline__ float2 ldg_r(const float2* p) { return __ldg(p); }
__device__ __forceinline__ double2 ldg_r(const double2* p) { return __ldg(p); }
__device__ __forceinline__ double4 ldg_r(const double4* p) {
    const double2 a = __ldg(reinterpret_cast<const double2*>(p)), b = __ldg(reinterpret_cast<const double2*>(p) + 1);
    return make_double4(a.x, a.y, b.x, b.y);
}
__device__ __forceinline__ float4 to_float4(float4 v)  { return v; }
__device__ __forceinline__ float4 to_float4(double4 v) { return make_float4((float)v.x, (float)v.y, (float)v.z, (float)v.w); }

// Neighbour predicate, R7 (bit-specified):
//   d_a = fl(x_i - x_j) - shift_a   (shift_a in {-L_a, 0, +L_a}: the minimum image; exact when 0)
//   r2  = fma(dz, dz, fma(dy, dy, fl(dx*dx)));   cut = fl(kh * fl(h_i + h_j));   hit <=> r2 < fl(cut*cut)
__device__ __forceinline__ float pair_r2(float dx, float dy, float dz) {
    return __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
}
__device__ __forceinline__ float pair_cut2(float kh, float hi, float hj) {
    float cut = __fmul_rn(kh, __fadd_rn(hi, hj));
    return __fmul_rn(cut, cut);
}

// The double build evaluates DESIGN.md R7 in double as the reference side states it (products and sums rounded one by
// one, cut = k * (0.5 * (h_i + h_j))), so that the sets stay bit-exact there too.
__device__ __forceinline__ double pair_r2(double dx, double dy, double dz) {
    return __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
}
__device__ __forceinline__ double pair_cut2(double ksup, double hi, double hj) {
    const double cut = __dmul_rn(ksup, __dmul_rn(0.5, __dadd_rn(hi, hj)));
    return __dmul_rn(cut, cut);
}
__device__ __forceinline__ float  rsub(float a, float b)   { return __fsub_rn(a, b); }
__device__ __forceinline__ double rsub(double a, double b) { return __dsub_rn(a, b); }

// Dimensionless kernel profile f(q) and f'(q); W = sigma h^-d f, dW/dr = sigma h^-(d+1) f'.
template <int KERNEL, int DIM, class T>
__device__ __forceinline__ void kernel_profile(T q, T& f, T& df) {
    if (KERNEL == SPH_KERNEL_CUBIC) {
        T t = T(2.0) - q;
        T inner_f  = rfma(q * q, rfma(T(0.75), q, T(-1.5)), T(1.0));    // 1 - 1.5 q^2 + 0.75 q^3
        T inner_df = q * rfma(T(2.25), q, T(-3.0));                     // -3 q + 2.25 q^2
        T outer_f  = T(0.25) * t * t * t;
        T outer_df = T(-0.75) * t * t;
        bool in = q < T(1.0);
        f  = in ? inner_f : outer_f;
        df = in ? inner_df : outer_df;
        if (q >= T(2.0)) { f = T(0.0); df = T(0.0); }
    } else if (KERNEL == SPH_KERNEL_QUINTIC) {
        T a = rmax(T(3.0) - q, T(0.0)), b = rmax(T(2.0) - q, T(0.0)), c = rmax(T(1.0) - q, T(0.0));
        T a2 = a * a, b2 = b * b, c2 = c * c;
        T a4 = a2 * a2, b4 = b2 * b2, c4 = c2 * c2;
        f  = rfma(T(15.0), c4 * c, rfma(T(-6.0), b4 * b, a4 * a));
        df = rfma(T(-75.0), c4, rfma(T(30.0), b4, T(-5.0) * a4));
    } else {
        T t = rmax(rfma(T(-0.5), q, T(1.0)), T(0.0));
        T t2 = t * t;
        if (DIM == 1) { f = t2 * t * rfma(T(1.5), q, T(1.0)); df = T(-3.0) * q * t2; }
        else          { f = t2 * t2 * rfma(T(2.0), q, T(1.0)); df = T(-5.0) * q * t2 * t; }
    }
}

// ---- packed f32x2 forms (sm_100 FADD2 / FMUL2 / FFMA2: one issue slot for two lanes of work).  The drains evaluate
// two neighbours of a particle at a time: .x and .y are the two neighbours.  Round-to-nearest, same results as the
// scalar forms.
__device__ __forceinline__ float2 pk(float a, float b) { return make_float2(a, b); }
__device__ __forceinline__ float2 pk1(float a) { return make_float2(a, a); }
__device__ __forceinline__ float2 add2(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 sub2(float2 a, float2 b) { return __fadd2_rn(a, make_float2(-b.x, -b.y)); }
__device__ __forceinline__ float2 mul2(float2 a, float2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ float2 max2(float2 a, float b) { return make_float2(fmaxf(a.x, b), fmaxf(a.y, b)); }
__device__ __forceinline__ float2 rcp2(float2 a) { return make_float2(rcp_approx(a.x), rcp_approx(a.y)); }

template <int KERNEL, int DIM>
__device__ __forceinline__ void kernel_profile2(float2 q, float2& f, float2& df) {
    if (KERNEL == SPH_KERNEL_CUBIC) {
        const float2 t = sub2(pk1(2.0f), q);
        const float2 qq = mul2(q, q);
        const float2 inner_f  = fma2(qq, fma2(pk1(0.75f), q, pk1(-1.5f)), pk1(1.0f));   // 1 - 1.5 q^2 + 0.75 q^3
        const float2 inner_df = mul2(q, fma2(pk1(2.25f), q, pk1(-3.0f)));               // -3 q + 2.25 q^2
        const float2 tt = mul2(t, t);
        const float2 outer_f  = mul2(mul2(pk1(0.25f), t), tt);
        const float2 outer_df = mul2(pk1(-0.75f), tt);
        f.x  = q.x < 1.0f ? inner_f.x : (q.x < 2.0f ? outer_f.x : 0.0f);
        f.y  = q.y < 1.0f ? inner_f.y : (q.y < 2.0f ? outer_f.y : 0.0f);
        df.x = q.x < 1.0f ? inner_df.x : (q.x < 2.0f ? outer_df.x : 0.0f);
        df.y = q.y < 1.0f ? inner_df.y : (q.y < 2.0f ? outer_df.y : 0.0f);
    } else if (KERNEL == SPH_KERNEL_QUINTIC) {
        const float2 a = max2(sub2(pk1(3.0f), q), 0.0f), b = max2(sub2(pk1(2.0f), q), 0.0f), c = max2(sub2(pk1(1.0f), q), 0.0f);
        const float2 a2 = mul2(a, a), b2 = mul2(b, b), c2 = mul2(c, c);
        const float2 a4 = mul2(a2, a2), b4 = mul2(b2, b2), c4 = mul2(c2, c2);
        f  = fma2(pk1(15.0f), mul2(c4, c), fma2(pk1(-6.0f), mul2(b4, b), mul2(a4, a)));
        df = fma2(pk1(-75.0f), c4, fma2(pk1(30.0f), b4, mul2(pk1(-5.0f), a4)));
    } else {
        const float2 t = max2(fma2(pk1(-0.5f), q, pk1(1.0f)), 0.0f);
        const float2 t2 = mul2(t, t);
        if (DIM == 1) { f = mul2(mul2(t2, t), fma2(pk1(1.5f), q, pk1(1.0f))); df = mul2(mul2(pk1(-3.0f), q), t2); }
        else          { f = mul2(mul2(t2, t2), fma2(pk1(2.0f), q, pk1(1.0f))); df = mul2(mul2(pk1(-5.0f), q), mul2(t2, t)); }
    }
}

// p/rho^2 of the gamma = 7 Tait EOS for two densities (same polynomial as eos7_p)
__device__ __forceinline__ float2 eos7_p_over_rho2_2(float2 rho, float rho0, float inv_rho0, float B) {
    const float2 t = mul2(sub2(rho, pk1(rho0)), pk1(inv_rho0));
    float2 s = fma2(t, pk1(1.0f), pk1(7.0f));
    s = fma2(t, s, pk1(21.0f)); s = fma2(t, s, pk1(35.0f)); s = fma2(t, s, pk1(35.0f)); s = fma2(t, s, pk1(21.0f)); s = fma2(t, s, pk1(7.0f));
    s = mul2(t, s);
    return mul2(mul2(pk1(B), s), rcp2(mul2(rho, rho)));
}

__host__ __device__ inline double kernel_sigma(int kernel, int dim) {
    const double pi = 3.141592653589793238462643383279502884;
    if (kernel == SPH_KERNEL_CUBIC)   return dim == 1 ? 2.0 / 3.0 : dim == 2 ? 10.0 / (7.0 * pi) : 1.0 / pi;
    if (kernel == SPH_KERNEL_QUINTIC) return dim == 1 ? 1.0 / 120.0 : dim == 2 ? 7.0 / (478.0 * pi) : 1.0 / (120.0 * pi);
    return dim == 1 ? 5.0 / 8.0 : dim == 2 ? 7.0 / (4.0 * pi) : 21.0 / (16.0 * pi);
}
__host__ __device__ inline double kernel_support(int kernel) { return kernel == SPH_KERNEL_QUINTIC ? 3.0 : 2.0; }

// Tait EOS, eq.6 (L122) / Listing 4 L393-400.
// In float, (rho/rho0)^gamma - 1 cancels catastrophically for a weakly compressible fluid (rho ~ rho0), so it
// is evaluated from t = (rho - rho0)/rho0 (the subtraction is exact for rho within a factor 2 of rho0):
//   gamma = 7:  (1+t)^7 - 1 = t (7 + 21 t + 35 t^2 + 35 t^3 + 21 t^4 + 7 t^5 + t^6)   (exact identity)
//   otherwise:  expm1(gamma * log1p(t))
__device__ __forceinline__ float  eos_general(float gamma, float t)   { return expm1f(gamma * log1pf(t)); }
__device__ __forceinline__ double eos_general(double gamma, double t) { return expm1(gamma * log1p(t)); }
template <class T>
__device__ __forceinline__ T eos_pressure(T rho, T rho0, T B, T gamma, int gamma_is_7) {
    const T t = (rho - rho0) / rho0;
    T s;
    if (gamma_is_7) s = t * rfma(t, rfma(t, rfma(t, rfma(t, rfma(t, rfma(t, T(1.0), T(7.0)), T(21.0)), T(35.0)), T(35.0)), T(21.0)), T(7.0));
    else s = eos_general(gamma, t);
    return B * s;
}

// p/rho^2 of the Tait EOS with gamma = 7 from rho alone (the momentum pair loop recomputes it per neighbour
// instead of gathering it): same polynomial as eos_pressure, t formed with a multiplication by 1/rho0.
template <class T>
__device__ __forceinline__ T eos7_p(T rho, T rho0, T inv_rho0, T B) {
    const T t = (rho - rho0) * inv_rho0;
    const T s = t * rfma(t, rfma(t, rfma(t, rfma(t, rfma(t, rfma(t, T(1.0), T(7.0)), T(21.0)), T(35.0)), T(35.0)), T(21.0)), T(7.0));
    return B * s;
}
template <class T>
__device__ __forceinline__ T eos7_p_over_rho2(T rho, T rho0, T inv_rho0, T B) {
    return eos7_p(rho, rho0, inv_rho0, B) * rcp_approx(rho * rho);
}

// Cell coordinate of a position on one axis (clamped; out-of-range on a non-periodic axis is flagged by the caller).
__device__ __forceinline__ int cell_coord(float x, float lo, float inv, int n) {
    int c = __float2int_rd((x - lo) * inv);
    return min(max(c, 0), n - 1);
}

