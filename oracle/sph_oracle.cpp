// ORACLE -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
// Plain, slow, fp64 CPU implementation of the SPH hot path of arXiv 1909.04504 (PySPH), written
// from PAPER.md.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
// legs may call it.  It shares no code, header, table or constant with the CUDA path
// (paper_1909_04504_b200/csrc) and neither includes the other.
//
// What each function follows (PAPER.md line, section / equation):
//   orc_W / orc_dWdr      kernel W(r,h), compact support W=0 for r>kh (L106, Sec.2).  The paper prints
//                         no kernel formula (L209, L435 "not shown here"): textbook forms, R1.
//   orc_neighbors         N(i) = { j : |x_i-x_j| < k h_ij } (L106, L158 Sec.2.2); brute force, or the
//                         linked-list cell grid of L163-166 (head[] / next[] over a flattened cell id).
//   orc_density           rho_i = sum_j m_j W_ij                          (eq.3)
//   orc_eos               p = B[(rho/rho0)^gamma - 1], B = rho0 c0^2/gamma (eq.6; Listing 4)
//   orc_accel             a_i += -m_j (p_i/rho_i^2 + p_j/rho_j^2 + Pi_ij) grad_i W_ij   (eq.8-9;
//                         Listing 4); Pi_ij = Monaghan artificial viscosity, R9
//                         (the paper only says "classic scheme of [36]", L185);
//                         arho_i += m_j (v_i-v_j).grad_i W_ij             (eq.7; Listing 4)
//   loop structure        for d_idx: for s_idx in neighbours(d_idx): loop(...)   (Listing 7)
//   orc_visc_laminar      a_i += m_j 4 nu/(rho_i+rho_j) (r_ij.grad_i W_ij)/(r^2 + eta h^2) u_ij     (eq.10)
// The integrators (eqs. 12-14; forward Euler, Fig.2) are per-particle arithmetic and live in
// sph_oracle.py.
//
// Readings: symmetric h_ij = (h_i+h_j)/2 (R3); strict '<' (R4); self pair included (R5);
// minimum image applied to the difference (R6); grad W := 0 at r = 0 (R18).
// Neighbour predicate: pred32 = 1 evaluates the DESIGN.md R7 float expression (the GPU decides set
// membership in float; both sides take that decision in the same precision); pred32 = 0 is the same
// expression in double.  Everything else is double.
//
// Parity pins: tests/test_oracle_*.py (kernel integrals, finite differences, lattice sums, brute force
// vs cell list, momentum conservation, continuum limits, Taylor-Green decay bracket, hand cases).
// UNPINNED: the *choice* of Pi_ij form and its constants, h_ij convention, rho stepping.
//
// Build: g++ -O2 -ffp-contract=off -fopenmp -shared -fPIC   (OpenMP over destinations: timing only)
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <vector>
#include <algorithm>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_API extern "C"

struct orc_domain {
    int dim;            // 2 or 3 (1 accepted by the kernel functions only)
    double lo[3], hi[3];
    int periodic[3];
};

enum { ORC_CUBIC = 0, ORC_QUINTIC = 1, ORC_WENDLAND_C2 = 2 };

// ---------------------------------------------------------------------------------------------
// Kernels.  q = r/h,  W = sigma_d h^-d f(q),  dW/dr = sigma_d h^-(d+1) f'(q).   DESIGN.md R1/R2.
// ---------------------------------------------------------------------------------------------
ORC_API double orc_support(int kernel) { return kernel == ORC_QUINTIC ? 3.0 : 2.0; }

static double sigma_of(int kernel, int dim) {
    const double pi = 3.14159265358979323846;
    if (kernel == ORC_CUBIC)   return dim == 1 ? 2.0 / 3.0 : dim == 2 ? 10.0 / (7.0 * pi) : 1.0 / pi;
    if (kernel == ORC_QUINTIC) return dim == 1 ? 1.0 / 120.0 : dim == 2 ? 7.0 / (478.0 * pi) : 1.0 / (120.0 * pi);
    /* Wendland C2 */          return dim == 1 ? 5.0 / 8.0 : dim == 2 ? 7.0 / (4.0 * pi) : 21.0 / (16.0 * pi);
}

static double f_of(int kernel, int dim, double q) {
    if (kernel == ORC_CUBIC) {
        if (q < 1.0) return 1.0 - 1.5 * q * q + 0.75 * q * q * q;
        if (q < 2.0) { double t = 2.0 - q; return 0.25 * t * t * t; }
        return 0.0;
    }
    if (kernel == ORC_QUINTIC) {
        if (q >= 3.0) return 0.0;
        double v = std::pow(3.0 - q, 5);
        if (q < 2.0) v -= 6.0 * std::pow(2.0 - q, 5);
        if (q < 1.0) v += 15.0 * std::pow(1.0 - q, 5);
        return v;
    }
    if (q >= 2.0) return 0.0;
    double t = 1.0 - 0.5 * q;
    if (dim == 1) return t * t * t * (1.5 * q + 1.0);
    return t * t * t * t * (2.0 * q + 1.0);
}

static double df_of(int kernel, int dim, double q) {
    if (kernel == ORC_CUBIC) {
        if (q < 1.0) return -3.0 * q + 2.25 * q * q;
        if (q < 2.0) { double t = 2.0 - q; return -0.75 * t * t; }
        return 0.0;
    }
    if (kernel == ORC_QUINTIC) {
        if (q >= 3.0) return 0.0;
        double v = -5.0 * std::pow(3.0 - q, 4);
        if (q < 2.0) v += 30.0 * std::pow(2.0 - q, 4);
        if (q < 1.0) v -= 75.0 * std::pow(1.0 - q, 4);
        return v;
    }
    if (q >= 2.0) return 0.0;
    double t = 1.0 - 0.5 * q;
    if (dim == 1) return -3.0 * q * t * t;
    return -5.0 * q * t * t * t;
}

ORC_API double orc_W(int kernel, int dim, double r, double h) {
    return sigma_of(kernel, dim) / std::pow(h, dim) * f_of(kernel, dim, r / h);
}
ORC_API double orc_dWdr(int kernel, int dim, double r, double h) {
    return sigma_of(kernel, dim) / std::pow(h, dim + 1) * df_of(kernel, dim, r / h);
}

// ---------------------------------------------------------------------------------------------
// Pair geometry.
// ---------------------------------------------------------------------------------------------
// minimum image on the difference (R6): d = xi - xj; if d > L/2: d -= L; else if d < -L/2: d += L
static inline double minimg64(double d, double L, int periodic) {
    if (periodic) { if (d > 0.5 * L) d -= L; else if (d < -0.5 * L) d += L; }
    return d;
}

// DESIGN.md R7, the specified float predicate (must be compiled with -ffp-contract=off):
//   d_a  = fl(x_i - x_j), then the minimum-image shift in float with L_a = (float)(hi_a - lo_a)
//   r2   = fmaf(dz, dz, fmaf(dy, dy, fl(dx*dx)))
//   cut  = fl( (float)(k/2) * fl(h_i + h_j) ),  cut2 = fl(cut*cut);   neighbour  <=>  r2 < cut2
static inline bool pred_float(const orc_domain* dom, double k,
                              double xi, double yi, double zi, double hi_,
                              double xj, double yj, double zj, double hj) {
    float d[3] = { (float)xi - (float)xj, (float)yi - (float)yj, (float)zi - (float)zj };
    for (int a = 0; a < 3; ++a) {
        if (a < dom->dim && dom->periodic[a]) {
            float L = (float)(dom->hi[a] - dom->lo[a]);
            float half = 0.5f * L;
            if (d[a] > half) d[a] = d[a] - L; else if (d[a] < -half) d[a] = d[a] + L;
        }
    }
    if (dom->dim < 3) d[2] = 0.0f;
    float r2 = fmaf(d[2], d[2], fmaf(d[1], d[1], d[0] * d[0]));
    float s = (float)hi_ + (float)hj;
    float cut = (float)(0.5 * k) * s;
    float cut2 = cut * cut;
    return r2 < cut2;
}

static inline bool pred_double(const orc_domain* dom, double k,
                               double xi, double yi, double zi, double hi_,
                               double xj, double yj, double zj, double hj) {
    double d[3] = { xi - xj, yi - yj, zi - zj };
    for (int a = 0; a < 3; ++a)
        d[a] = (a < dom->dim) ? minimg64(d[a], dom->hi[a] - dom->lo[a], dom->periodic[a]) : 0.0;
    double r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
    double cut = k * (0.5 * (hi_ + hj));
    return r2 < cut * cut;
}

struct Pts { int64_t n; const double *x, *y, *z, *h; };

static inline bool is_nb(const orc_domain* dom, double k, int pred32, const Pts& D, int64_t i, const Pts& S, int64_t j) {
    double zi = dom->dim == 3 ? D.z[i] : 0.0, zj = dom->dim == 3 ? S.z[j] : 0.0;
    return pred32 ? pred_float(dom, k, D.x[i], D.y[i], zi, D.h[i], S.x[j], S.y[j], zj, S.h[j])
                  : pred_double(dom, k, D.x[i], D.y[i], zi, D.h[i], S.x[j], S.y[j], zj, S.h[j]);
}

// ---------------------------------------------------------------------------------------------
// Linked-list cell grid over the SOURCE particles (flattened 1-D cell id ->
// head[], per-particle next[]; cells of size = the (maximum) support radius, L158-160).
// ---------------------------------------------------------------------------------------------
struct CellGrid {
    int dim; int n[3]; double lo[3], inv[3]; int periodic[3];
    std::vector<int64_t> head, next;
    int cell_of(int a, double x) const {
        int c = (int)std::floor((x - lo[a]) * inv[a]);
        if (c < 0) c = 0; if (c >= n[a]) c = n[a] - 1;
        return c;
    }
};

static void build_grid(CellGrid& g, const orc_domain* dom, double k, const Pts& D, const Pts& S) {
    double hmax = 0.0;
    for (int64_t i = 0; i < D.n; ++i) hmax = std::max(hmax, D.h[i]);
    for (int64_t j = 0; j < S.n; ++j) hmax = std::max(hmax, S.h[j]);
    double cell = k * hmax * (1.0 + 1e-6);        // >= every pair cut-off k*h_ij, with slack for the float predicate
    if (!(cell > 0.0)) cell = 1.0;
    g.dim = dom->dim;
    const double* dc[3] = { D.x, D.y, D.z };
    const double* sc[3] = { S.x, S.y, S.z };
    for (int a = 0; a < 3; ++a) {
        g.periodic[a] = (a < dom->dim) ? dom->periodic[a] : 0;
        if (a >= dom->dim) { g.n[a] = 1; g.lo[a] = 0.0; g.inv[a] = 0.0; continue; }
        double lo, hi;
        if (g.periodic[a]) { lo = dom->lo[a]; hi = dom->hi[a]; }
        else {                                    // own bounding box: independent of the caller's domain box
            lo = 1e300; hi = -1e300;
            for (int64_t i = 0; i < D.n; ++i) { lo = std::min(lo, dc[a][i]); hi = std::max(hi, dc[a][i]); }
            for (int64_t j = 0; j < S.n; ++j) { lo = std::min(lo, sc[a][j]); hi = std::max(hi, sc[a][j]); }
            if (lo > hi) { lo = 0.0; hi = 1.0; }
            hi += 1e-9 * std::max(1.0, std::fabs(hi)) + 1e-300;
        }
        double L = hi - lo;
        int n = (int)std::floor(L / cell);
        if (n < 1) n = 1;
        if (g.periodic[a] && n < 3) n = 1;        // fewer than 3 cells: stencil would alias, use one cell
        if (n > 2048) n = 2048;                   // bound the head[] size; cells only get larger (still correct)
        g.n[a] = n; g.lo[a] = lo; g.inv[a] = n / L;
    }
    int64_t nc = (int64_t)g.n[0] * g.n[1] * g.n[2];
    g.head.assign(nc, -1);
    g.next.assign(S.n, -1);
    for (int64_t j = S.n - 1; j >= 0; --j) {
        int c[3] = { g.cell_of(0, S.x[j]), g.dim > 1 ? g.cell_of(1, S.y[j]) : 0, g.dim > 2 ? g.cell_of(2, S.z[j]) : 0 };
        int64_t id = ((int64_t)c[2] * g.n[1] + c[1]) * g.n[0] + c[0];
        g.next[j] = g.head[id]; g.head[id] = j;
    }
}

// the 3^d neighbouring boxes of the query particle's cell (L158, Fig.1), de-duplicated
static int stencil_axis(const CellGrid& g, int a, int c, int out[3]) {
    int cnt = 0;
    for (int o = -1; o <= 1; ++o) {
        int cc = c + o;
        if (g.periodic[a]) cc = ((cc % g.n[a]) + g.n[a]) % g.n[a];
        else if (cc < 0 || cc >= g.n[a]) continue;
        bool dup = false;
        for (int t = 0; t < cnt; ++t) dup |= (out[t] == cc);
        if (!dup) out[cnt++] = cc;
    }
    return cnt;
}

// Calls visit(j) for every source j passing the predicate for destination i (ascending j for brute force).
template <class F>
static inline void for_neighbors(const orc_domain* dom, double k, int pred32, int method, const CellGrid* g,
                                 const Pts& D, int64_t i, const Pts& S, F visit) {
    if (method == 0) {
        for (int64_t j = 0; j < S.n; ++j) if (is_nb(dom, k, pred32, D, i, S, j)) visit(j);
        return;
    }
    int cx[3], cy[3], cz[3];
    int nx = stencil_axis(*g, 0, g->cell_of(0, D.x[i]), cx);
    int ny = g->dim > 1 ? stencil_axis(*g, 1, g->cell_of(1, D.y[i]), cy) : (cy[0] = 0, 1);
    int nz = g->dim > 2 ? stencil_axis(*g, 2, g->cell_of(2, D.z[i]), cz) : (cz[0] = 0, 1);
    for (int c = 0; c < nz; ++c) for (int b = 0; b < ny; ++b) for (int a = 0; a < nx; ++a) {
        int64_t id = ((int64_t)cz[c] * g->n[1] + cy[b]) * g->n[0] + cx[a];
        for (int64_t j = g->head[id]; j >= 0; j = g->next[j])
            if (is_nb(dom, k, pred32, D, i, S, j)) visit(j);
    }
}

// ---------------------------------------------------------------------------------------------
// Neighbour sets as CSR, each row sorted ascending.  Returns the total count; fills `indices` only
// when cap >= total.  offsets has nd+1 entries.
// ---------------------------------------------------------------------------------------------
ORC_API int64_t orc_neighbors(const orc_domain* dom, double k, int pred32, int method,
                      int64_t nd, const double* xd, const double* yd, const double* zd, const double* hd,
                      int64_t ns, const double* xs, const double* ys, const double* zs, const double* hs,
                      int64_t* offsets, int64_t* indices, int64_t cap) {
    Pts D{nd, xd, yd, zd, hd}, S{ns, xs, ys, zs, hs};
    CellGrid g; if (method) build_grid(g, dom, k, D, S);
    std::vector<int64_t> cnt(nd + 1, 0);
    #pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < nd; ++i) {
        int64_t c = 0;
        for_neighbors(dom, k, pred32, method, &g, D, i, S, [&](int64_t) { ++c; });
        cnt[i] = c;
    }
    offsets[0] = 0;
    for (int64_t i = 0; i < nd; ++i) offsets[i + 1] = offsets[i] + cnt[i];
    int64_t total = offsets[nd];
    if (indices && cap >= total) {
        #pragma omp parallel for schedule(dynamic, 64)
        for (int64_t i = 0; i < nd; ++i) {
            int64_t* row = indices + offsets[i]; int64_t c = 0;
            for_neighbors(dom, k, pred32, method, &g, D, i, S, [&](int64_t j) { row[c++] = j; });
            std::sort(row, row + c);
        }
    }
    return total;
}

// ---------------------------------------------------------------------------------------------
// Fields.  Each call handles ONE (dest array, source array) pair and ACCUMULATES into its outputs, so
// the caller runs "all the fluid neighbours ... and then the solid neighbours" (L423-425, L528-534)
// after the initialize() values (0, or gravity: L408-411) have been stored.
// abs_* (nullable) receive sum_j |term|: the forward-error scale of the sum.
// ---------------------------------------------------------------------------------------------
struct PairGeom { double d[3]; double r; double hij; };

static inline PairGeom geom64(const orc_domain* dom, const double* xd, const double* yd, const double* zd, const double* hd,
                              int64_t i, const double* xs, const double* ys, const double* zs, const double* hs, int64_t j) {
    PairGeom g;
    g.d[0] = minimg64(xd[i] - xs[j], dom->hi[0] - dom->lo[0], dom->periodic[0]);
    g.d[1] = minimg64(yd[i] - ys[j], dom->hi[1] - dom->lo[1], dom->periodic[1]);
    g.d[2] = dom->dim == 3 ? minimg64(zd[i] - zs[j], dom->hi[2] - dom->lo[2], dom->periodic[2]) : 0.0;
    g.r = std::sqrt(g.d[0] * g.d[0] + g.d[1] * g.d[1] + g.d[2] * g.d[2]);
    g.hij = 0.5 * (hd[i] + hs[j]);
    return g;
}

// eq.3 (L112): rho_i += sum_j m_j W(x_i - x_j, h_ij)
ORC_API void orc_density(const orc_domain* dom, int kernel, int pred32, int method,
                 int64_t nd, const double* xd, const double* yd, const double* zd, const double* hd,
                 int64_t ns, const double* xs, const double* ys, const double* zs, const double* hs, const double* ms,
                 double* rho, double* abs_rho, int64_t* n_pairs) {
    double k = orc_support(kernel);
    Pts D{nd, xd, yd, zd, hd}, S{ns, xs, ys, zs, hs};
    CellGrid g; if (method) build_grid(g, dom, k, D, S);
    int64_t pairs = 0;
    #pragma omp parallel for schedule(dynamic, 64) reduction(+:pairs)
    for (int64_t i = 0; i < nd; ++i) {
        double acc = 0.0; int64_t c = 0;
        for_neighbors(dom, k, pred32, method, &g, D, i, S, [&](int64_t j) {
            PairGeom pg = geom64(dom, xd, yd, zd, hd, i, xs, ys, zs, hs, j);
            acc += ms[j] * orc_W(kernel, dom->dim, pg.r, pg.hij);
            ++c;
        });
        rho[i] += acc;                       // every term is >= 0, so abs-sum == sum
        if (abs_rho) abs_rho[i] += acc;
        pairs += c;
    }
    if (n_pairs) *n_pairs += pairs;
}

// eq.6 (L122), Listing 4:  B = rho0*c0*c0/gamma;  p = B*(pow(rho/rho0, gamma) - 1.0)
ORC_API void orc_eos(int64_t n, const double* rho, double rho0, double c0, double gamma, double* p) {
    double B = rho0 * c0 * c0 / gamma;
    for (int64_t i = 0; i < n; ++i) p[i] = B * (std::pow(rho[i] / rho0, gamma) - 1.0);
}

// eq.8-9 (L128-132) + artificial viscosity Pi_ij (R9) + eq.7 (L126):
//   grad_i W_ij = dW/dr(r, h_ij) * (x_i - x_j)/r          (:= 0 at r = 0, R18)
//   Pi_ij = -alpha * c0 * mu_ij / rhobar_ij  if v_ij.r_ij < 0 else 0,
//           mu_ij = h_ij (v_ij.r_ij) / (r^2 + eps h_ij^2),  rhobar_ij = (rho_i + rho_j)/2
//   a_i   += -m_j (p_i/rho_i^2 + p_j/rho_j^2 + Pi_ij) grad_i W_ij        (Listing 4)
//   arho_i += m_j (v_i - v_j) . grad_i W_ij                              (Listing 4)
ORC_API void orc_accel(const orc_domain* dom, int kernel, double alpha, double eps, double c0, int pred32, int method,
               int64_t nd, const double* xd, const double* yd, const double* zd,
               const double* ud, const double* vd, const double* wd,
               const double* hd, const double* rhod, const double* pd,
               int64_t ns, const double* xs, const double* ys, const double* zs,
               const double* us, const double* vs, const double* ws,
               const double* hs, const double* ms, const double* rhos, const double* ps,
               double* au, double* av, double* aw, double* arho,
               double* abs_a, double* abs_arho, double* visc_power, int64_t* n_pairs) {
    double k = orc_support(kernel);
    Pts D{nd, xd, yd, zd, hd}, S{ns, xs, ys, zs, hs};
    CellGrid g; if (method) build_grid(g, dom, k, D, S);
    int64_t pairs = 0;
    #pragma omp parallel for schedule(dynamic, 64) reduction(+:pairs)
    for (int64_t i = 0; i < nd; ++i) {
        double sx = 0, sy = 0, sz = 0, sr = 0, sabs = 0, srabs = 0, spow = 0; int64_t c = 0;
        double pri = pd[i] / (rhod[i] * rhod[i]);
        for_neighbors(dom, k, pred32, method, &g, D, i, S, [&](int64_t j) {
            ++c;
            PairGeom pg = geom64(dom, xd, yd, zd, hd, i, xs, ys, zs, hs, j);
            if (pg.r == 0.0) return;                               // R18: grad W = 0 (self pair)
            double dw = orc_dWdr(kernel, dom->dim, pg.r, pg.hij);
            double gx = dw * pg.d[0] / pg.r, gy = dw * pg.d[1] / pg.r, gz = dw * pg.d[2] / pg.r;   // DWIJ
            double vx = ud[i] - us[j], vy = vd[i] - vs[j];                                         // VIJ
            double vz = dom->dim == 3 ? wd[i] - ws[j] : 0.0;
            double vr = vx * pg.d[0] + vy * pg.d[1] + vz * pg.d[2];
            double Pi = 0.0;
            if (vr < 0.0) {
                double mu = pg.hij * vr / (pg.r * pg.r + eps * pg.hij * pg.hij);
                double rhobar = 0.5 * (rhod[i] + rhos[j]);
                Pi = -alpha * c0 * mu / rhobar;
            }
            double tmp = pri + ps[j] / (rhos[j] * rhos[j]) + Pi;
            sx += -ms[j] * tmp * gx; sy += -ms[j] * tmp * gy; sz += -ms[j] * tmp * gz;
            sabs += std::fabs(ms[j] * (std::fabs(pri) + std::fabs(ps[j] / (rhos[j] * rhos[j])) + std::fabs(Pi)) * dw);
            spow += -ms[j] * Pi * (gx * ud[i] + gy * vd[i] + gz * (dom->dim == 3 ? wd[i] : 0.0));
            double vdw = vx * gx + vy * gy + vz * gz;
            sr += ms[j] * vdw; srabs += std::fabs(ms[j] * vdw);
        });
        au[i] += sx; av[i] += sy; if (aw) aw[i] += sz;
        if (arho) arho[i] += sr;
        if (abs_a) abs_a[i] += sabs;
        if (abs_arho) abs_arho[i] += srabs;
        if (visc_power) visc_power[i] += spow;   // u_i . a_visc,i (per unit mass), for the dissipation pins
        pairs += c;
    }
    if (n_pairs) *n_pairs += pairs;
}

// Laminar viscosity, eq.10 (L134-136), added to the accelerations when nu != 0:
//   a_visc,i = sum_j m_j 4 nu / (rho_i + rho_j) * (r_ij . grad_i W_ij) / (|r_ij|^2 + eta h_ij^2) * u_ij
// (h in the regulariser read as h_ij, R3).  visc_power accumulates u_i . a_visc,i for the dissipation pin.
ORC_API void orc_visc_laminar(const orc_domain* dom, int kernel, double nu, double eta, int pred32, int method,
               int64_t nd, const double* xd, const double* yd, const double* zd,
               const double* ud, const double* vd, const double* wd, const double* hd, const double* rhod,
               int64_t ns, const double* xs, const double* ys, const double* zs,
               const double* us, const double* vs, const double* ws,
               const double* hs, const double* ms, const double* rhos,
               double* au, double* av, double* aw, double* abs_a, double* visc_power) {
    double k = orc_support(kernel);
    Pts D{nd, xd, yd, zd, hd}, S{ns, xs, ys, zs, hs};
    CellGrid g; if (method) build_grid(g, dom, k, D, S);
    #pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < nd; ++i) {
        double sx = 0, sy = 0, sz = 0, sabs = 0;
        for_neighbors(dom, k, pred32, method, &g, D, i, S, [&](int64_t j) {
            PairGeom pg = geom64(dom, xd, yd, zd, hd, i, xs, ys, zs, hs, j);
            if (pg.r == 0.0) return;                               // R18: grad W = 0
            double dw = orc_dWdr(kernel, dom->dim, pg.r, pg.hij);
            double rdw = dw * pg.r;                                // r_ij . grad_i W_ij = dW/dr * r
            double vx = ud[i] - us[j], vy = vd[i] - vs[j];
            double vz = dom->dim == 3 ? wd[i] - ws[j] : 0.0;
            double c = ms[j] * 4.0 * nu / (rhod[i] + rhos[j]) * rdw / (pg.r * pg.r + eta * pg.hij * pg.hij);
            sx += c * vx; sy += c * vy; sz += c * vz;
            sabs += std::fabs(c) * std::sqrt(vx * vx + vy * vy + vz * vz);
        });
        au[i] += sx; av[i] += sy; if (aw) aw[i] += sz;
        if (abs_a) abs_a[i] += sabs;
        if (visc_power) visc_power[i] += sx * ud[i] + sy * vd[i] + (dom->dim == 3 ? sz * wd[i] : 0.0);
    }
}

ORC_API int orc_num_threads(void) {          // threads the OpenMP loops above actually use (bench cpu_baseline "cores")
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

ORC_API void orc_set_num_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

