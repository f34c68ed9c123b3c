// C ABI of libsph_b200.so (include/sph.h): argument checking, workspace, and the order of kernels.
// Every step of the path runs in the kernels of sph_nnps.cu / sph_density.cu / sph_accel.cu; this file only
// marshals arguments and enqueues launches.  There is no CPU fallback.
#include "sph_ctx.cuh"
#include <math.h>
#include <string.h>
#include <stdlib.h>
#include <new>

static const int N_STAGE_FIELDS = 14;


extern "C" const char* sph_strerror(int code) {
    switch (code) {
        case SPH_OK: return "ok";
        case SPH_ERR_NULL: return "null pointer";
        case SPH_ERR_BAD_ARG: return "bad argument";
        case SPH_ERR_CAPACITY: return "capacity exceeded";
        case SPH_ERR_STALE_NNPS: return "no neighbour structure: call sph_nnps_build first";
        case SPH_ERR_OUT_OF_DOMAIN: return "particles outside a non-periodic domain";
        case SPH_ERR_NONFINITE: return "non-finite value produced";
        case SPH_ERR_CUDA: return "CUDA error";
    }
    return "unknown error";
}
extern "C" const char* sph_last_error(const sph_ctx* c) { return c ? c->err : "null context"; }
extern "C" int sph_abi_version(void) { return SPH_ABI_VERSION; }
extern "C" int sph_real_size(void) { return (int)sizeof(sph_real); }

static void drop_graph(sph_ctx* c) {
    if (c->step_graph) { cudaGraphExecDestroy(c->step_graph); c->step_graph = nullptr; }
}

static void default_tables(sph_ctx* c) {
    uint32_t all = (1u << c->na) - 1u, dyn = 0;
    for (int a = 0; a < c->na; ++a) if (!c->fixed[a]) dyn |= 1u << a;
    for (int a = 0; a < SPH_MAX_ARRAYS; ++a) {
        const bool live = a < c->na;
        c->tbl_density[a] = live ? all : 0u;
        c->tbl_accel[a] = (live && !c->fixed[a]) ? all : 0u;
        c->tbl_arho[a] = live ? (c->fixed[a] ? dyn : all) : 0u;     // Listing 3
    }
}

static void set_consts(sph_ctx* c) {
    const sph_params& P = c->prm;
    PairConsts& pc = c->pc;
    memset(&pc, 0, sizeof(pc));
    pc.kh = (real)(0.5 * kernel_support(P.kernel));
    pc.ksup = (real)kernel_support(P.kernel);
    pc.sigma = (real)kernel_sigma(P.kernel, c->dom.dim);
    pc.rho0 = (real)P.rho0;
    pc.B = (real)(P.rho0 * P.c0 * P.c0 / P.gamma);
    pc.gamma = (real)P.gamma;
    pc.gamma_is_7 = (P.gamma == 7.0);
    pc.visc = (real)(-2.0 * P.alpha * P.c0);
    pc.eps = (real)P.eps;
    pc.nu4 = (real)(4.0 * P.nu); pc.eta = (real)P.eta;
    for (int k = 0; k < 3; ++k) pc.g[k] = (real)P.g[k];
    pc.all_mask = (1u << c->na) - 1u;
    pc.h_const = 1; pc.hinv_const = 1; pc.fac_const = 1;
}

extern "C" int sph_create(sph_ctx** out, const sph_params* params, const sph_domain* domain,
                          int n_arrays, const int64_t* capacity, void* cuda_stream) {
    if (!out || !params || !domain || !capacity) return SPH_ERR_NULL;
    *out = nullptr;
    if (n_arrays < 1 || n_arrays > SPH_MAX_ARRAYS) return SPH_ERR_BAD_ARG;
    if (domain->dim != 2 && domain->dim != 3) return SPH_ERR_BAD_ARG;
    if (params->kernel < 0 || params->kernel > SPH_KERNEL_WENDLAND_C2) return SPH_ERR_BAD_ARG;
    if (!(params->rho0 > 0) || !(params->c0 > 0) || !(params->gamma > 0)) return SPH_ERR_BAD_ARG;
    if (params->xsub < 0 || params->xsub > 16) return SPH_ERR_BAD_ARG;
    if (params->levels < 0 || params->levels > SPH_MAX_LEVELS) return SPH_ERR_BAD_ARG;
    if (params->integrator != SPH_INTEGRATOR_PC && params->integrator != SPH_INTEGRATOR_EULER) return SPH_ERR_BAD_ARG;
    if (!(params->nu >= 0) || !(params->eta >= 0)) return SPH_ERR_BAD_ARG;
    for (int k = 0; k < domain->dim; ++k) if (!(domain->hi[k] > domain->lo[k])) return SPH_ERR_BAD_ARG;
    int64_t tot = 0;
    for (int a = 0; a < n_arrays; ++a) {
        if (capacity[a] < 0 || capacity[a] > (int64_t)SPH_META_IDX_MASK) return SPH_ERR_BAD_ARG;
        tot += capacity[a];
    }
    if (tot > (int64_t)0x7fffff00) return SPH_ERR_BAD_ARG;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return SPH_ERR_CUDA;   // no CPU fallback

    sph_ctx* c = new (std::nothrow) sph_ctx;
    if (!c) return SPH_ERR_CUDA;
    memset(c, 0, sizeof(*c));
    c->stream = (cudaStream_t)cuda_stream;
    c->prm = *params; c->dom = *domain; c->na = n_arrays;
    if (domain->dim == 2) { c->dom.lo[2] = 0; c->dom.hi[2] = 1; c->dom.periodic[2] = 0; }
    for (int a = 0; a < n_arrays; ++a) c->cap[a] = capacity[a];
    c->cap_total = tot;
    default_tables(c);
    set_consts(c);
    c->xsub = params->xsub ? params->xsub : 6;
    const int nl_slots = params->nlist_slots ? params->nlist_slots : 192;
    *out = c;                                  // so the caller can read sph_last_error / destroy on failure
    SPH_CUDA_OK(c, cudaGetDevice(&c->device));
    SPH_CUDA_OK(c, cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, c->device));

    const size_t N = (size_t)tot + 1;
    c->max_keys = 8 * tot + 65536; if (c->max_keys > ((int64_t)1 << 27)) c->max_keys = (int64_t)1 << 27;
    for (int b = 0; b < 2; ++b) {
        SPH_CUDA_OK(c, cudaMalloc(&c->S[b].posh, N * sizeof(real4)));
        SPH_CUDA_OK(c, cudaMalloc(&c->S[b].velm, N * sizeof(real4)));
        SPH_CUDA_OK(c, cudaMalloc(&c->S[b].rp, N * sizeof(real2)));
        SPH_CUDA_OK(c, cudaMalloc(&c->S[b].meta, N * sizeof(uint32_t)));
        SPH_CUDA_OK(c, cudaMalloc(&c->S[b].cell, N * sizeof(uint32_t)));
    }
    for (int b = 0; b < 2; ++b) SPH_CUDA_OK(c, cudaMalloc(&c->S[b].acc, N * sizeof(real4)));
    SPH_CUDA_OK(c, cudaMalloc(&c->key, (N + 1) * sizeof(uint32_t)));
    SPH_CUDA_OK(c, cudaMalloc(&c->rank, (N + 1) * sizeof(uint32_t)));
    SPH_CUDA_OK(c, cudaMalloc(&c->cell_count, (size_t)(c->max_keys + 2) * sizeof(uint32_t)));
    SPH_CUDA_OK(c, cudaMalloc(&c->cell_start, (size_t)(c->max_keys + 2) * sizeof(uint32_t)));
    const size_t scan_n = (size_t)(c->max_keys > tot ? c->max_keys : tot) + 2;
    SPH_CUDA_OK(c, cudaMalloc(&c->scan_state, (scan_n / 2048 + 4) * sizeof(unsigned long long)));
    SPH_CUDA_OK(c, cudaMemsetAsync(c->scan_state, 0, (scan_n / 2048 + 4) * sizeof(unsigned long long), c->stream));
    c->scan_tiles_cap = (int)(scan_n / 4096 + 2);
    SPH_CUDA_OK(c, cudaMalloc(&c->scan_tiles, 2 * (size_t)(c->scan_tiles_cap + 1) * sizeof(uint32_t)));
    SPH_CUDA_OK(c, cudaMalloc(&c->scan_ticket, 2 * sizeof(uint32_t)));
    SPH_CUDA_OK(c, cudaMemsetAsync(c->scan_ticket, 0, 2 * sizeof(uint32_t), c->stream));
    SPH_CUDA_OK(c, cudaMalloc(&c->staging, N * N_STAGE_FIELDS * sizeof(real)));
    SPH_CUDA_OK(c, cudaMalloc(&c->counters, CNT_COUNT * sizeof(unsigned long long)));
    SPH_CUDA_OK(c, cudaMalloc(&c->hminmax, 4 * sizeof(long long)));
    if (nl_slots > 0 && tot > 0) {
        const size_t warps = (size_t)(tot + 31) / 32;
        size_t rows = warps * (size_t)nl_slots + 64;      // + slack: a replaying warp always fetches a whole block image (26 rows)
        if (rows > 0xfffffff0ull) rows = 0xfffffff0ull;
        c->nl.pool_rows = (uint32_t)(rows - 32);          // rows the recorder may hand out; the last 32 are only ever over-read
        SPH_CUDA_OK(c, cudaMalloc(&c->nl.pool, rows * 32 * sizeof(uint32_t)));
        SPH_CUDA_OK(c, cudaMalloc(&c->nl.head, (warps + 2) * sizeof(uint32_t)));
        c->nl.used = (uint32_t*)(c->counters + CNT_NL_USED);
    }
    SPH_CUDA_OK(c, cudaMemsetAsync(c->counters, 0, CNT_COUNT * sizeof(unsigned long long), c->stream));
    for (int b = 0; b < 2; ++b) SPH_CUDA_OK(c, cudaMemsetAsync(c->S[b].acc, 0, N * sizeof(real4), c->stream));
    SPH_CUDA_OK(c, cudaStreamSynchronize(c->stream));
    return SPH_OK;
}

extern "C" int sph_destroy(sph_ctx* c) {
    if (!c) return SPH_ERR_NULL;
    cudaStreamSynchronize(c->stream);
    for (int b = 0; b < 2; ++b) {
        cudaFree(c->S[b].posh); cudaFree(c->S[b].velm); cudaFree(c->S[b].rp); cudaFree(c->S[b].meta); cudaFree(c->S[b].cell);
    }
    cudaFree(c->S[0].acc); cudaFree(c->S[1].acc); cudaFree(c->key); cudaFree(c->rank); cudaFree(c->cell_count); cudaFree(c->cell_start);
    cudaFree(c->nl.pool); cudaFree(c->nl.head);
    cudaFree(c->scan_state); cudaFree(c->scan_ticket); cudaFree(c->scan_tiles); cudaFree(c->staging); cudaFree(c->counters); cudaFree(c->hminmax);
    if (c->step_graph) cudaGraphExecDestroy(c->step_graph);
    for (int k = 0; k < c->prof_cap; ++k) { cudaEventDestroy(c->prof[k].a); cudaEventDestroy(c->prof[k].b); }
    free(c->prof);
    delete c;
    return SPH_OK;
}

extern "C" int sph_set_tables(sph_ctx* c, const uint32_t* density_src, const uint32_t* accel_src, const uint32_t* arho_src) {
    if (!c) return SPH_ERR_NULL;
    const uint32_t all = (1u << c->na) - 1u;
    const uint32_t* in[3] = { density_src, accel_src, arho_src };
    uint32_t* dst[3] = { c->tbl_density, c->tbl_accel, c->tbl_arho };
    for (int t = 0; t < 3; ++t) if (in[t]) for (int a = 0; a < c->na; ++a) if (in[t][a] & ~all) return sph_fail(c, SPH_ERR_BAD_ARG, "source mask names a non-existent array");
    for (int t = 0; t < 3; ++t) if (in[t]) for (int a = 0; a < c->na; ++a) dst[t][a] = in[t][a];
    c->tables_user = true;
    drop_graph(c);
    return SPH_OK;
}

// Level grids.  One level when h is constant: cell >= k*h_max (L158-160) with a margin that absorbs the float
// rounding of the cell coordinate.  When h varies the particles are binned into geometric h classes (ratio <= ~1.6
// per level) and every level gets its own grid with cell >= k * (largest h of the level): the paper's remedy for
// "cells become too large" (L158-160, L171) without giving up the sort-by-cell-key structure.
static int size_grid(sph_ctx* c) {
    GridDesc& g = c->grid;
    memset(&g, 0, sizeof(g));
    g.dim = c->dom.dim; g.na = c->na;
    const double ksup = kernel_support(c->prm.kernel);
    if (!((double)c->h_max > 0.0)) return sph_fail(c, SPH_ERR_BAD_ARG, "h_max must be positive");
    double big = 0.0;
    for (int k = 0; k < 3; ++k) {
        g.per[k] = (k < g.dim) ? (c->dom.periodic[k] != 0) : 0;
        g.lo[k] = (float)c->dom.lo[k]; g.hi[k] = (float)c->dom.hi[k];
        g.L[k] = (float)(c->dom.hi[k] - c->dom.lo[k]);
        g.Lr[k] = sizeof(real) == 8 ? (real)(c->dom.hi[k] - c->dom.lo[k]) : (real)g.L[k];
        g.lor[k] = (real)c->dom.lo[k]; g.hir[k] = (real)c->dom.hi[k];
        if (k < g.dim) big = fmax(big, fmax(fmax(fabs(c->dom.lo[k]), fabs(c->dom.hi[k])), c->dom.hi[k] - c->dom.lo[k]));
    }
    g.uabs = (float)(1.1920929e-7 * big);
    const double ratio = (double)c->h_max / (double)c->h_min;
    int nlev = 1;
    if (c->variable_h) {
        nlev = c->prm.levels > 0 ? c->prm.levels : (int)ceil(log(ratio) / log(1.6) - 1.0e-9);
        nlev = nlev < 1 ? 1 : (nlev > SPH_MAX_LEVELS ? SPH_MAX_LEVELS : nlev);
    }
    int xsub = c->xsub;
    double scale = 1.0;
    for (int iter = 0; iter < 96; ++iter) {
        int64_t total = 0; bool ok = true;
        for (int l = 0; l < nlev && ok; ++l) {
            LevelDesc& Lv = g.lev[l];
            // every h of level l is <= hmax_l (float thresholds; level_of_h uses the same comparisons on both sides)
            const float hmax_f = (float)c->h_max;           // float(h) <= float(h_max) for every h (monotone rounding): the search runs in float
            Lv.hmax = (l == nlev - 1) ? hmax_f : (float)((double)c->h_min * pow(ratio, (l + 1.0) / nlev));
            if (l == nlev - 1 || Lv.hmax > hmax_f) Lv.hmax = hmax_f;
            const double cutoff = ksup * (double)Lv.hmax;
            int64_t cells = 1;
            for (int k = 0; k < 3; ++k) {
                const double L = (k < g.dim) ? c->dom.hi[k] - c->dom.lo[k] : 1.0;
                int n = 1;
                if (k < g.dim) {
                    const double est = L / (cutoff * scale);
                    const double margin = 1.0e-3 + 4.0e-7 * est;
                    double nd = floor(L / (cutoff * scale * (1.0 + margin)));
                    if (nd > 1.0e6) nd = 1.0e6;
                    n = nd < 1.0 ? 1 : (int)nd;
                    if (g.per[k] && n < 3) {
                        if (scale > 1.0) { ok = false; break; }      // cannot coarsen further
                        return sph_fail(c, SPH_ERR_BAD_ARG, "a periodic axis needs at least 3 cells of size k*h_max");
                    }
                }
                if (k == 0) n *= xsub;
                Lv.nc[k] = n;
                Lv.inv_cell[k] = (float)(n / L);
                cells *= n;
            }
            Lv.xsub = xsub;
            Lv.base = (uint32_t)total;
            total += cells;
            if (total > ((int64_t)1 << 30)) ok = false;
        }
        g.nlev = nlev;
        if (ok && total * c->na <= c->max_keys) { c->n_keys = total * c->na; g.cells_total = (uint32_t)total; g.n_sorted = (uint32_t)c->n_total; g.dbg = c->counters; return SPH_OK; }
        if (xsub > 1) xsub /= 2; else if (nlev > 1) --nlev; else scale *= 1.26;
    }
    return sph_fail(c, SPH_ERR_CAPACITY, "cell table too small for this domain / h_max");
}

static real* stage_field(sph_ctx* c, int field, int array) { return c->staging + ((size_t)field * (c->cap_total + 1) + c->base[array]); }

extern "C" int sph_nnps_build(sph_ctx* c, int n_arrays, const sph_array* arrays) {
    if (!c || !arrays) return SPH_ERR_NULL;
    if (n_arrays != c->na) return sph_fail(c, SPH_ERR_BAD_ARG, "n_arrays differs from sph_create");
    c->built = false; c->have_accel = false; c->have_arho = false; c->nl_valid = false;
    c->counters_fresh = false; c->heads_fresh = false;
    drop_graph(c);
    int64_t tot = 0;
    bool all_acc = true, all_arho = true, any_p = false;
    for (int a = 0; a < c->na; ++a) {
        const sph_array& A = arrays[a];
        if (A.n < 0) return sph_fail(c, SPH_ERR_BAD_ARG, "negative n");
        if (A.n > c->cap[a]) return sph_fail(c, SPH_ERR_CAPACITY, "array larger than its capacity");
        if (A.n > 0 && (!A.x || !A.y || !A.h || (c->dom.dim == 3 && !A.z))) return sph_fail(c, SPH_ERR_NULL, "x, y, (z), h are required");
        if (A.mem != SPH_MEM_DEVICE && A.mem != SPH_MEM_HOST) return sph_fail(c, SPH_ERR_BAD_ARG, "bad mem");
        c->n[a] = A.n; c->base[a] = tot; c->fixed[a] = (A.flags & SPH_ARRAY_FIXED) ? 1 : 0;
        tot += A.n;
        if (A.n > 0 && !c->fixed[a] && (!A.ax || !A.ay || (c->dom.dim == 3 && !A.az))) all_acc = false;
        if (A.n > 0 && !A.arho) all_arho = false;
        if (A.n > 0 && A.p) any_p = true;
    }
    c->base[c->na] = tot; c->n_total = tot;
    if (!c->tables_user) default_tables(c);

    PackArgs P; memset(&P, 0, sizeof(P));
    P.na = c->na;
    for (int a = 0; a <= c->na; ++a) P.base[a] = c->base[a];
    for (int a = 0; a < c->na; ++a) {
        const sph_array& A = arrays[a];
        const real* src[N_STAGE_FIELDS] = { A.x, A.y, A.z, A.u, A.v, A.w, A.h, A.m, A.rho, A.p, A.ax, A.ay, A.az, A.arho };
        const real* use[N_STAGE_FIELDS];
        for (int f = 0; f < N_STAGE_FIELDS; ++f) {
            use[f] = src[f];
            if (A.mem == SPH_MEM_HOST && src[f] && A.n > 0) {
                real* d = stage_field(c, f, a);
                SPH_CUDA_OK(c, cudaMemcpyAsync(d, src[f], (size_t)A.n * sizeof(real), cudaMemcpyHostToDevice, c->stream));
                use[f] = d;
            }
        }
        P.a[a] = PackSrc{ use[0], use[1], use[2], use[3], use[4], use[5], use[6], use[7], use[8], use[9],
                          use[10], use[11], use[12], use[13] };
    }
    SPH_CUDA_OK(c, cudaMemsetAsync(c->counters, 0, CNT_COUNT * sizeof(unsigned long long), c->stream));
    c->cur = 0;
    int rc = nnps_pack(c, P); if (rc) return rc;
    long long hmm[4] = { 0, 0, 0, 0 };                  // ordered-integer images of h min/max, |m| min/max (int or long long words)
    SPH_CUDA_OK(c, cudaMemcpyAsync(hmm, c->hminmax, 4 * (sizeof(real) == 8 ? sizeof(long long) : sizeof(int)), cudaMemcpyDeviceToHost, c->stream));
    SPH_CUDA_OK(c, cudaStreamSynchronize(c->stream));
    real hm[4];
    for (int k = 0; k < 4; ++k) memcpy(&hm[k], (const char*)hmm + k * sizeof(real), sizeof(real));
    if (tot == 0) {                            // no particles at all: any grid will do; size it so that a periodic box gets its >= 3 cells
        double minL = 1.0e300;
        for (int k = 0; k < c->dom.dim; ++k) minL = fmin(minL, c->dom.hi[k] - c->dom.lo[k]);
        c->h_min = c->h_max = (real)(minL / (4.0 * kernel_support(c->prm.kernel)));
    }
    else { c->h_min = hm[0]; c->h_max = hm[1]; }
    if (!(c->h_max > 0) || !isfinite((double)c->h_max)) return sph_fail(c, SPH_ERR_BAD_ARG, "smoothing lengths must be positive and finite");
    c->variable_h = (c->h_min != c->h_max);
    c->p_is_eos = !any_p;
    c->pc.uniform_m = (tot > 0 && !c->variable_h && hm[2] == hm[3]) ? 1 : 0;
    c->pc.varh_um = (tot > 0 && c->variable_h && hm[2] == hm[3] && c->p_is_eos && c->pc.gamma_is_7) ? 1 : 0;
    c->pc.m_const = hm[3];
    c->pc.h_const = c->h_max;
    c->pc.hinv_const = (real)(1.0 / (double)c->h_max);
    c->pc.fac_const = (real)(kernel_sigma(c->prm.kernel, c->dom.dim) / pow((double)c->h_max, c->dom.dim));
    rc = size_grid(c); if (rc) return rc;
    SPH_CUDA_OK(c, cudaMemsetAsync(c->cell_count, 0, (size_t)(c->n_keys + 1) * sizeof(uint32_t), c->stream));   // once per build; k_scan re-clears it
    rc = nnps_key_hist(c); if (rc) return rc;
    rc = nnps_sort_from_keys(c, true); if (rc) return rc;
    c->built = true; c->steps_done = 0;
    c->have_accel = all_acc && tot > 0; c->have_arho = all_arho && tot > 0;     // restart from caller-supplied a^n
    return SPH_OK;
}

// caller-order output of up to 12 fields of one array, to device pointers or through the staging buffer to host
static int emit(sph_ctx* c, int array, OutPtrs O, int mem) {
    real** f = (real**)&O;
    const int NF = sizeof(OutPtrs) / sizeof(real*);
    const size_t n = (size_t)c->n[array];
    if (mem == SPH_MEM_DEVICE) return nnps_gather_out(c, array, O);
    real* host[NF]; int used = 0;
    for (int k = 0; k < NF; ++k) { host[k] = f[k]; if (f[k]) { if (used >= N_STAGE_FIELDS) return sph_fail(c, SPH_ERR_BAD_ARG, "too many host outputs in one call"); f[k] = c->staging + (size_t)used * (c->cap_total + 1); ++used; } }
    int rc = nnps_gather_out(c, array, O); if (rc) return rc;
    for (int k = 0; k < NF; ++k) if (host[k] && n) SPH_CUDA_OK(c, cudaMemcpyAsync(host[k], f[k], n * sizeof(real), cudaMemcpyDeviceToHost, c->stream));
    SPH_CUDA_OK(c, cudaStreamSynchronize(c->stream));
    return SPH_OK;
}

static int zero_counters(sph_ctx* c, int first, int last) {       // one memset for counters [first, last]
    SPH_CUDA_OK(c, cudaMemsetAsync(c->counters + first, 0, (size_t)(last - first + 1) * sizeof(unsigned long long), c->stream));
    return SPH_OK;
}

// one search per sorted order, shared by every pair pass that follows (no-op without a record pool)
static int ensure_search(sph_ctx* c) {
    if (c->nl_valid || c->nl.pool == nullptr) return SPH_OK;
    return launch_search(c);
}

extern "C" int sph_summation_density(sph_ctx* c, int dest, uint32_t source_mask, sph_real* rho_out, sph_real* p_out, int mem) {
    if (!c) return SPH_ERR_NULL;
    if (!c->built) return sph_fail(c, SPH_ERR_STALE_NNPS, sph_strerror(SPH_ERR_STALE_NNPS));
    if (dest < 0 || dest >= c->na || source_mask == 0 || (source_mask & ~c->pc.all_mask)) return sph_fail(c, SPH_ERR_BAD_ARG, "bad dest / source_mask");
    uint32_t masks[SPH_MAX_ARRAYS] = { 0, 0, 0, 0 };
    masks[dest] = source_mask;
    int rc = ensure_search(c); if (rc) return rc;
    rc = zero_counters(c, CNT_PAIRS_DENSITY, CNT_CAND_DENSITY); if (rc) return rc;
    rc = launch_density(c, masks); if (rc) return rc;
    if (rho_out || p_out) { OutPtrs O; memset(&O, 0, sizeof(O)); O.rho = rho_out; O.p = p_out; return emit(c, dest, O, mem); }
    return SPH_OK;
}

extern "C" int sph_wcsph_accel(sph_ctx* c, int dest, uint32_t source_mask, sph_real* ax, sph_real* ay, sph_real* az, sph_real* arho, int mem) {
    if (!c) return SPH_ERR_NULL;
    if (!c->built) return sph_fail(c, SPH_ERR_STALE_NNPS, sph_strerror(SPH_ERR_STALE_NNPS));
    if (dest < 0 || dest >= c->na || source_mask == 0 || (source_mask & ~c->pc.all_mask)) return sph_fail(c, SPH_ERR_BAD_ARG, "bad dest / source_mask");
    uint32_t masks[SPH_MAX_ARRAYS] = { 0, 0, 0, 0 };
    masks[dest] = source_mask;
    int rc = ensure_search(c); if (rc) return rc;
    rc = zero_counters(c, CNT_PAIRS_ACCEL, CNT_CAND_ACCEL); if (rc) return rc;
    const AccelRoles roles = { 0u, 0u, 0u, 0u };
    rc = launch_accel(c, masks, arho != nullptr, roles); if (rc) return rc;
    if (ax || ay || az || arho) { OutPtrs O; memset(&O, 0, sizeof(O)); O.ax = ax; O.ay = ay; O.az = az; O.arho = arho; return emit(c, dest, O, mem); }
    return SPH_OK;
}

// One evaluation F(x,u,rho) in group order (Listing 3): [density ->] EOS on all arrays | barrier |
// continuity + momentum.  Destinations that share a source mask share a launch.
static int evaluate(sph_ctx* c, bool continuity) {
    int rc;
    rc = ensure_search(c); if (rc) return rc;
    if (!c->counters_fresh) { rc = zero_counters(c, CNT_PAIRS_DENSITY, CNT_CAND_ACCEL); if (rc) return rc; }   // (k_update clears them inside a step)
    c->counters_fresh = false;
    auto grouped = [&](const uint32_t* tbl, const bool* take, auto&& fn) -> int {
        bool done[SPH_MAX_ARRAYS] = { false, false, false, false };
        for (int a = 0; a < c->na; ++a) {
            if (done[a] || !take[a] || !tbl[a]) continue;
            uint32_t masks[SPH_MAX_ARRAYS] = { 0, 0, 0, 0 };
            for (int b = a; b < c->na; ++b) if (!done[b] && take[b] && tbl[b] == tbl[a]) { masks[b] = tbl[b]; done[b] = true; }
            int r = fn(masks); if (r) return r;
        }
        return SPH_OK;
    };
    bool all[SPH_MAX_ARRAYS] = { true, true, true, true };
    if (!continuity) {
        rc = grouped(c->tbl_density, all, [&](const uint32_t* m) { return launch_density(c, m); });
        if (rc) return rc;
    }
    bool fused[SPH_MAX_ARRAYS], plain[SPH_MAX_ARRAYS], only[SPH_MAX_ARRAYS];
    // arrays whose acc.xyz / acc.w NO launch of this evaluation computes get zeros from the first launch (the sort
    // does not carry acc along: what lies in their rows belongs to other particles)
    AccelRoles first = { 0u, 0u, 0u, 0u };
    uint32_t keep = 0u;
    for (int a = 0; a < SPH_MAX_ARRAYS; ++a) {
        const bool acc = a < c->na && c->tbl_accel[a] != 0;
        const bool same = acc && continuity && c->tbl_arho[a] == c->tbl_accel[a];
        fused[a] = same; plain[a] = acc && !same;
        only[a] = a < c->na && continuity && c->tbl_arho[a] != 0 && !same;
        if (a < c->na && !acc) first.zero_xyz |= 1u << a;
        if (a < c->na && !(continuity && c->tbl_arho[a] != 0)) first.zero_w |= 1u << a;
        if (plain[a]) keep |= 1u << a;
    }
    bool launched = false;
    auto accel = [&](const uint32_t* m, bool want_arho, uint32_t arho_only, bool after_plain) -> int {
        AccelRoles r = { arho_only, after_plain ? (arho_only & keep) : 0u, launched ? 0u : first.zero_xyz, launched ? 0u : first.zero_w };
        launched = true;
        return launch_accel(c, m, want_arho, r);
    };
    // continuity mode: when no array needs two different source sets, ONE launch serves them all (fluid: momentum +
    // continuity from {fluid, solid}; solid: continuity only from {fluid}; the per-lane source mask filters)
    bool one = continuity;
    for (int a = 0; a < c->na; ++a) if (plain[a] && only[a]) one = false;
    if (one) {
        uint32_t masks[SPH_MAX_ARRAYS] = { 0, 0, 0, 0 }, ao = 0u; bool any = false;
        for (int a = 0; a < c->na; ++a) {
            if (fused[a] || plain[a]) masks[a] = c->tbl_accel[a];
            else if (only[a]) { masks[a] = c->tbl_arho[a]; ao |= 1u << a; }
            any = any || masks[a] != 0u;
        }
        if (any) { rc = accel(masks, true, ao, false); if (rc) return rc; }
    } else {
        rc = grouped(c->tbl_accel, fused, [&](const uint32_t* m) { return accel(m, true, 0u, false); }); if (rc) return rc;
        rc = grouped(c->tbl_accel, plain, [&](const uint32_t* m) { return accel(m, false, 0u, false); }); if (rc) return rc;
        rc = grouped(c->tbl_arho, only, [&](const uint32_t* m) {
            uint32_t ao = 0u; for (int a = 0; a < c->na; ++a) if (m[a]) ao |= 1u << a;
            return accel(m, true, ao, true); }); if (rc) return rc;
    }
    if (!launched && c->n_total > 0)      // no momentum / continuity destination at all: every acceleration is zero
        SPH_CUDA_OK(c, cudaMemsetAsync(c->S[c->cur].acc, 0, (size_t)c->n_total * sizeof(real4), c->stream));
    return SPH_OK;
}

// one step of the loop of sph_pc_step.   PC: (14 of the previous step) + 12 + 13 + key.   Euler: x += dt u ; u += dt a ;
// rho += dt arho ; key.   Then the sort (NNPS rebuilt every step, L443) and the evaluation.
static int step_body(sph_ctx* c, real dt, bool cont, bool kick2) {
    int rc = nnps_update_key_hist(c, dt, kick2, true, cont, true); if (rc) return rc;
    rc = nnps_sort_from_keys(c, false); if (rc) return rc;
    rc = evaluate(c, cont); if (rc) return rc;
    c->have_arho = cont;
    return SPH_OK;
}

// Captures TWO consecutive middle steps (the state buffers flip every step, so two steps return to the same
// buffers) into a CUDA graph: long runs of small problems are bound by launch latency, not by work.
static bool ensure_step_graph(sph_ctx* c, real dt, bool cont, bool kick2) {
    if (c->graph_off) return false;
    if (c->step_graph && c->graph_dt == dt && c->graph_cont == (cont ? 1 : 0) && c->graph_cur == c->cur) return true;
    drop_graph(c);
    const int64_t l0 = c->launches;
    cudaGraph_t graph = nullptr;
    if (cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) { cudaGetLastError(); c->graph_off = true; return false; }
    int rc = step_body(c, dt, cont, kick2);
    if (!rc) rc = step_body(c, dt, cont, kick2);
    const cudaError_t e = cudaStreamEndCapture(c->stream, &graph);
    c->graph_nodes = (int)(c->launches - l0);
    c->launches = l0;                                   // nothing ran: the captured launches are counted per replay
    if (rc || e != cudaSuccess || !graph) { if (graph) cudaGraphDestroy(graph); cudaGetLastError(); c->graph_off = true; return false; }
    const cudaError_t e2 = cudaGraphInstantiate(&c->step_graph, graph, 0);
    cudaGraphDestroy(graph);
    if (e2 != cudaSuccess) { c->step_graph = nullptr; cudaGetLastError(); c->graph_off = true; return false; }
    c->graph_dt = dt; c->graph_cont = cont ? 1 : 0; c->graph_cur = c->cur;
    return true;
}

extern "C" int sph_pc_step(sph_ctx* c, double dt, int n_steps, int density_mode) {
    if (!c) return SPH_ERR_NULL;
    if (!c->built) return sph_fail(c, SPH_ERR_STALE_NNPS, sph_strerror(SPH_ERR_STALE_NNPS));
    if (n_steps < 0 || (density_mode != SPH_DENSITY_SUMMATION && density_mode != SPH_DENSITY_CONTINUITY) || !isfinite(dt))
        return sph_fail(c, SPH_ERR_BAD_ARG, "bad n_steps / density_mode / dt");
    const bool cont = density_mode == SPH_DENSITY_CONTINUITY;
    int rc;
    if (!c->have_accel || (cont && !c->have_arho)) {                                             // a^0 = F(x^0, u^0)
        rc = evaluate(c, cont); if (rc) return rc; c->have_accel = true; c->have_arho = cont;
    }
    const bool euler = c->prm.integrator == SPH_INTEGRATOR_EULER;
    int s = 0;
    if (n_steps > 0) { rc = step_body(c, (real)dt, cont, false); if (rc) return rc; c->steps_done++; s = 1; }
    // long runs: replay a captured pair of steps (same kernels, same arguments, one graph launch per two steps)
    if (n_steps - s >= 8 && !c->prof_on && c->n_total > 0 && ensure_step_graph(c, (real)dt, cont, !euler)) {
        while (n_steps - s >= 2) {
            SPH_CUDA_OK(c, cudaGraphLaunch(c->step_graph, c->stream));
            c->launches += c->graph_nodes; c->steps_done += 2; s += 2;
        }
    }
    for (; s < n_steps; ++s) { rc = step_body(c, (real)dt, cont, !euler); if (rc) return rc; c->steps_done++; }
    if (n_steps > 0 && !euler) { rc = nnps_update_key_hist(c, (real)dt, true, false, cont, false); if (rc) return rc; }   // eq.14
    return SPH_OK;
}

extern "C" int sph_sync_state(sph_ctx* c, int array, const sph_array* out) {
    if (!c || !out) return SPH_ERR_NULL;
    if (!c->built) return sph_fail(c, SPH_ERR_STALE_NNPS, sph_strerror(SPH_ERR_STALE_NNPS));
    if (array < 0 || array >= c->na) return sph_fail(c, SPH_ERR_BAD_ARG, "bad array");
    if (out->n != c->n[array]) return sph_fail(c, SPH_ERR_CAPACITY, "out->n differs from the array size");
    OutPtrs O; memset(&O, 0, sizeof(O));
    O.x = out->x; O.y = out->y; O.z = out->z; O.u = out->u; O.v = out->v; O.w = out->w; O.rho = out->rho; O.p = out->p;
    O.ax = out->ax; O.ay = out->ay; O.az = out->az; O.arho = out->arho;
    return emit(c, array, O, out->mem);
}

extern "C" int sph_get_accel(sph_ctx* c, int array, sph_real* ax, sph_real* ay, sph_real* az, sph_real* arho, int mem) {
    if (!c) return SPH_ERR_NULL;
    if (!c->built) return sph_fail(c, SPH_ERR_STALE_NNPS, sph_strerror(SPH_ERR_STALE_NNPS));
    if (array < 0 || array >= c->na) return sph_fail(c, SPH_ERR_BAD_ARG, "bad array");
    OutPtrs O; memset(&O, 0, sizeof(O)); O.ax = ax; O.ay = ay; O.az = az; O.arho = arho;
    return emit(c, array, O, mem);
}

extern "C" int sph_nnps_get_neighbors(sph_ctx* c, int dest, int src, int64_t* offsets, int32_t* indices,
                                      int64_t cap, int64_t* total, int mem) {
    if (!c || !offsets || !total) return SPH_ERR_NULL;
    if (!c->built) return sph_fail(c, SPH_ERR_STALE_NNPS, sph_strerror(SPH_ERR_STALE_NNPS));
    if (dest < 0 || dest >= c->na || src < 0 || src >= c->na) return sph_fail(c, SPH_ERR_BAD_ARG, "bad dest / src");
    return nnps_export_neighbors(c, dest, src, offsets, indices, cap, total, mem);
}

extern "C" int sph_stencil_candidates(sph_ctx* c, int64_t* out) {
    if (!c || !out) return SPH_ERR_NULL;
    if (!c->built) return sph_fail(c, SPH_ERR_STALE_NNPS, sph_strerror(SPH_ERR_STALE_NNPS));
    return nnps_stencil_candidates(c, out);
}

static int read_counters(sph_ctx* c, unsigned long long* h) {
    SPH_CUDA_OK(c, cudaMemcpyAsync(h, c->counters, CNT_COUNT * sizeof(unsigned long long), cudaMemcpyDeviceToHost, c->stream));
    SPH_CUDA_OK(c, cudaStreamSynchronize(c->stream));
    return SPH_OK;
}

extern "C" int sph_synchronize(sph_ctx* c) {
    if (!c) return SPH_ERR_NULL;
    unsigned long long h[CNT_COUNT];
    int rc = read_counters(c, h); if (rc) return rc;
    if (h[CNT_OUT_OF_DOMAIN]) { snprintf(c->err, sizeof(c->err), "%llu particle updates fell outside the non-periodic domain box", h[CNT_OUT_OF_DOMAIN]); return SPH_ERR_OUT_OF_DOMAIN; }
    if (h[CNT_NONFINITE]) { snprintf(c->err, sizeof(c->err), "%llu non-finite results", h[CNT_NONFINITE]); return SPH_ERR_NONFINITE; }
    if (h[CNT_ASSERT]) { snprintf(c->err, sizeof(c->err), "%llu device-side bounds assertions failed (SPH_DEBUG_ASSERT build)", h[CNT_ASSERT]); return SPH_ERR_CUDA; }
    return SPH_OK;
}

extern "C" int sph_get_stats(sph_ctx* c, sph_stats* out) {
    if (!c || !out) return SPH_ERR_NULL;
    unsigned long long h[CNT_COUNT];
    int rc = read_counters(c, h); if (rc) return rc;
    memset(out, 0, sizeof(*out));
    const LevelDesc& top = c->grid.lev[c->grid.nlev > 0 ? c->grid.nlev - 1 : 0];    // the coarsest level: cells >= k h_max
    for (int k = 0; k < 3; ++k) {
        out->n_cells[k] = top.nc[k];
        out->cell_size[k] = top.nc[k] ? (c->dom.hi[k] - c->dom.lo[k]) / top.nc[k] : 0.0;
    }
    out->n_levels = c->grid.nlev;
    out->n_keys = c->n_keys;
    out->n_particles = c->n_total;
    out->pairs_density = (int64_t)h[CNT_PAIRS_DENSITY];
    out->pairs_accel = (int64_t)h[CNT_PAIRS_ACCEL];
    out->candidates_density = (int64_t)h[CNT_CAND_DENSITY];
    out->candidates_accel = (int64_t)h[CNT_CAND_ACCEL];
    out->candidates_search = (int64_t)h[CNT_CAND_SEARCH];
    out->candidates = out->candidates_density + out->candidates_accel + out->candidates_search;
    out->kernel_launches = c->launches;
    out->steps_done = c->steps_done;
    out->variable_h = c->variable_h ? 1 : 0;
    out->h_max = (float)c->h_max;
    out->xsub = top.xsub;
    out->used_rows = c->last_used_rows ? 1 : 0;
    out->nlist_rows_capacity = c->nl.pool_rows;
    out->nlist_fallback_warps = (int64_t)h[CNT_OVERFLOW];
    if (c->nl.used) {
        uint32_t u = 0;
        SPH_CUDA_OK(c, cudaMemcpyAsync(&u, c->nl.used, sizeof(u), cudaMemcpyDeviceToHost, c->stream));
        SPH_CUDA_OK(c, cudaStreamSynchronize(c->stream));
        out->nlist_rows_used = u;
    }
    return SPH_OK;
}

// ---- per-kernel device timing ----------------------------------------------------------------------
static const int PROF_MAX = 1 << 15;

int sph_prof_begin(sph_ctx* c, int id) {
    if (c->prof_used >= PROF_MAX) { c->prof_dropped++; return -1; }
    if (c->prof_used >= c->prof_cap) {
        const int ncap = c->prof_cap ? c->prof_cap * 2 : 256;
        sph_ctx::ProfRec* np = (sph_ctx::ProfRec*)realloc(c->prof, (size_t)ncap * sizeof(sph_ctx::ProfRec));
        if (!np) { c->prof_dropped++; return -1; }
        c->prof = np;
        for (int k = c->prof_cap; k < ncap; ++k) {
            if (cudaEventCreate(&c->prof[k].a) != cudaSuccess || cudaEventCreate(&c->prof[k].b) != cudaSuccess) { c->prof_cap = k; c->prof_dropped++; return -1; }
        }
        c->prof_cap = ncap;
    }
    const int r = c->prof_used++;
    c->prof[r].id = id;
    cudaEventRecord(c->prof[r].a, c->stream);
    return r;
}
void sph_prof_end(sph_ctx* c, int rec) { cudaEventRecord(c->prof[rec].b, c->stream); }

extern "C" int sph_set_profiling(sph_ctx* c, int enable) {
    if (!c) return SPH_ERR_NULL;
    SPH_CUDA_OK(c, cudaStreamSynchronize(c->stream));
    c->prof_on = enable != 0; c->prof_used = 0; c->prof_dropped = 0;
    return SPH_OK;
}

extern "C" int sph_get_profile(sph_ctx* c, sph_profile* out) {
    if (!c || !out) return SPH_ERR_NULL;
    SPH_CUDA_OK(c, cudaStreamSynchronize(c->stream));
    memset(out, 0, sizeof(*out));
    for (int r = 0; r < c->prof_used; ++r) {
        float ms = 0.0f;
        SPH_CUDA_OK(c, cudaEventElapsedTime(&ms, c->prof[r].a, c->prof[r].b));
        const int id = c->prof[r].id;
        if (id >= 0 && id < SPH_K_COUNT) { out->launches[id]++; out->ms[id] += (double)ms; }
    }
    out->dropped = c->prof_dropped;
    return SPH_OK;
}

extern "C" const char* sph_kernel_name(int id) {
    switch (id) {
        case SPH_K_PACK: return "k_pack";
        case SPH_K_KEY: return "k_key_hist";
        case SPH_K_UPDATE: return "k_update";
        case SPH_K_SCAN: return "k_scan";
        case SPH_K_SCAN_REDUCE: return "k_scan_reduce";
        case SPH_K_SCAN_TILES: return "k_scan_tiles";
        case SPH_K_SCATTER: return "k_scatter";
        case SPH_K_DENSITY: return "k_density";
        case SPH_K_ACCEL: return "k_accel";
        case SPH_K_OUTPUT: return "k_gather_out";
        case SPH_K_NEIGHBORS: return "k_neighbors";
        case SPH_K_ACCEL_LIST: return "k_accel_list";
        case SPH_K_SEARCH: return "k_search";
        case SPH_K_DENSITY_LIST: return "k_density_list";
        case SPH_K_UPDATE_KICK: return "k_update_kick";
    }
    return "";
}
