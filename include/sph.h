/* sph.h -- C ABI of the B200-native SPH hot path of arXiv 1909.04504 (PySPH).
 *
 * One library, libsph_b200.so, hand-written CUDA for sm_100a.  Every step of the path runs in its
 * kernels; there is NO CPU fallback: each call fails with SPH_ERR_CUDA if no device is usable.
 *
 * Problem statement (PAPER.md, cited as L<line>):
 *   - particles live in NAMED ARRAYS of per-particle properties x,y,z,u,v,w,h,m,rho,p, one 1-D
 *     contiguous array per property (L205, L316);
 *   - an equation acts on ONE destination array from a LIST of source arrays (L382, L423-425);
 *   - neighbours of i are the particles within the kernel support k*h (L106, L158), found with a
 *     uniform cell grid sorted by cell key, rebuilt whenever particles move (L158-170, L443);
 *   - groups are barriers: the EOS of ALL arrays completes before the momentum equation (L337).
 *
 * Conventions
 *   real type      sph_real = float (the paper's GPU runs are single precision, L733): libsph_b200.so.  The same sources
 *                  built with -DSPH_REAL_DOUBLE give libsph_b200_f64.so with sph_real = double (north_star: "1e-12
 *                  for an fp64 build flag"): the same calls, every particle buffer in double; sph_real_size() tells
 *                  which one was loaded.  There the neighbour search still runs in float on float-rounded positions
 *                  (it is conservative), the exact predicate and all field arithmetic in double.
 *   pointers       every particle buffer is CALLER-OWNED.  `mem` says where it lives: SPH_MEM_DEVICE
 *                  (device pointers on the context's device) or SPH_MEM_HOST (host pointers; the library
 *                  copies through its own staging buffers with cudaMemcpyAsync on the context stream --
 *                  pinned memory makes those copies asynchronous).  The library never frees or
 *                  reallocates caller memory.  Arrays must be contiguous; z,w may be NULL when dim == 2.
 *   ownership      sph_ctx is opaque and LIBRARY-OWNED; it holds all workspace (cell tables, the
 *                  cell-sorted mirror of the particle state), allocated once in sph_create from
 *                  `capacity`.  No call of the path allocates device memory after sph_create; the one exception is
 *                  the verification export sph_nnps_get_neighbors with HOST pointers, which allocates and frees two
 *                  temporary device buffers for its result.
 *   asynchrony     all work is enqueued on the stream given to sph_create.  Calls marked [sync]
 *                  synchronise that stream before returning; the others do not.
 *   errors         every call returns 0 (SPH_OK) or a negative sph_error.  Argument errors are detected
 *                  on the host before any work is enqueued.  Device-side conditions (a particle outside a
 *                  non-periodic domain, a non-finite result) set a device flag that the next [sync] call
 *                  reports.  sph_last_error(ctx) gives a message.  n == 0 arrays are legal.
 *   order          results are returned in the CALLER's particle order (the internal state is cell-sorted).
 */
#ifndef SPH_B200_H
#define SPH_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#ifdef SPH_REAL_DOUBLE
typedef double sph_real;
#else
typedef float sph_real;
#endif

#define SPH_MAX_ARRAYS 4
#define SPH_ABI_VERSION 5

typedef struct sph_ctx sph_ctx;

enum sph_error {
    SPH_OK = 0,
    SPH_ERR_NULL = -1,          /* a required pointer is NULL                                  */
    SPH_ERR_BAD_ARG = -2,       /* invalid value (dim, kernel, mask, periodic axis with < 3 cells ...) */
    SPH_ERR_CAPACITY = -3,      /* n exceeds the capacity given to sph_create, or an output is too small */
    SPH_ERR_STALE_NNPS = -4,    /* call needs a neighbour structure and none has been built      */
    SPH_ERR_OUT_OF_DOMAIN = -5, /* [sync] particles left a non-periodic domain box               */
    SPH_ERR_NONFINITE = -6,     /* [sync] NaN/Inf produced by a pair loop                        */
    SPH_ERR_CUDA = -7           /* CUDA runtime error (message in sph_last_error)                */
};

enum sph_kernel {               /* smoothing kernels, R1 (the paper prints none: L209, L435) */
    SPH_KERNEL_CUBIC = 0,       /* cubic spline,   support 2h */
    SPH_KERNEL_QUINTIC = 1,     /* quintic spline, support 3h */
    SPH_KERNEL_WENDLAND_C2 = 2  /* Wendland C2,    support 2h */
};

enum sph_density_mode {
    SPH_DENSITY_SUMMATION = 0,  /* rho from eq.3 (L112) every evaluation                          */
    SPH_DENSITY_CONTINUITY = 1  /* rho integrated from eq.7 (L126), as the paper's dam break (L142, L369-374) */
};

enum sph_integrator {
    SPH_INTEGRATOR_PC = 0,      /* predictor-corrector, eqs. 12-14 (L148-152), R10 (default)             */
    SPH_INTEGRATOR_EULER = 1    /* forward Euler, the paper's worked example (L335, Fig.2), R22:
                                   x += dt u ; u += dt a ; rho += dt arho, all from the values of step n        */
};

enum sph_mem { SPH_MEM_DEVICE = 0, SPH_MEM_HOST = 1 };
enum sph_array_flags { SPH_ARRAY_DYNAMIC = 0, SPH_ARRAY_FIXED = 1 /* x,u never updated (tank walls, L142) */ };

typedef struct sph_domain {     /* create_domain / update_domain (L443-445) */
    int dim;                    /* 2 or 3 */
    double lo[3], hi[3];        /* box; on a non-periodic axis it must enclose all particles */
    int periodic[3];            /* per axis; a periodic axis needs (hi-lo) >= 3 * k * h_max */
} sph_domain;

typedef struct sph_params {
    int kernel;                 /* enum sph_kernel */
    double rho0, c0, gamma;     /* Tait EOS, eq.6 (L122): p = (rho0 c0^2/gamma)[(rho/rho0)^gamma - 1] */
    double alpha, eps;          /* artificial viscosity (R9): Pi = -alpha c0 mu/rhobar, mu = h vr/(r^2+eps h^2) */
    double g[3];                /* body force = initial value of the accumulator (Listing 4) */
    int move;                   /* 1: sph_pc_step applies eq.13 (default); 0: positions frozen (config C5) */
    double nu, eta;             /* laminar viscosity, eq.10 (L134-136): a_i += sum_j m_j 4 nu/(rho_i+rho_j)
                                 * (r_ij . grad_i W_ij)/(r_ij^2 + eta h_ij^2) u_ij, in the same pair loop as eq.9.
                                 * nu = 0 (default): term off.  eta: the paper's regulariser (0.01 is customary) */
    int integrator;             /* enum sph_integrator: what sph_pc_step steps with */
    /* Tuning knobs of the neighbour search; results do not depend on them (0 = default). */
    int xsub;                   /* x sub-cells per support radius (1..16; default 0 = 6)                           */
    int levels;                 /* variable h: number of h classes, each with its own cell grid (PAPER.md L158-160,
                                 * L171: one grid sized by h_max "becomes inefficient"); 0 = as many as keep the h ratio
                                 * of a class <= ~1.6 (at most 8); 1 = the paper's single grid sized by h_max      */
    int nlist_slots;            /* record pool of the pair passes, in rows of 32 words per warp (32 particles) of
                                 * capacity (default 192, i.e. 768 B per particle of capacity; < 0: no pool, every
                                 * pair pass searches itself).  ONE search per sorted order records one 32-bit
                                 * candidate mask per particle and batch of 32 candidates; the density and momentum
                                 * passes that follow replay them (and apply the exact predicate).  A warp whose
                                 * masks do not fit is searched again by the pair passes
                                 * (sph_stats.nlist_fallback_warps counts them). */
} sph_params;

typedef struct sph_array {      /* one named particle array (L316) */
    int64_t n;
    int flags;                  /* enum sph_array_flags */
    int mem;                    /* enum sph_mem: where the pointers below live */
    sph_real *x, *y, *z;        /* positions      (z NULL allowed when dim == 2) */
    sph_real *u, *v, *w;        /* velocities     (w NULL allowed when dim == 2; all NULL -> 0) */
    sph_real *h;                /* smoothing length; sets the search radius (L316) */
    sph_real *m;                /* mass           (NULL -> 0: array only queries, never a source of mass) */
    sph_real *rho;              /* density        (NULL -> rho0) */
    sph_real *p;                /* pressure       (NULL -> EOS(rho)) */
    sph_real *ax, *ay, *az, *arho; /* accelerations of the last evaluation: the paper's au, av, aw, arho properties
                                 * (L402-418).  Input to sph_nnps_build (restart: if every dynamic array gives
                                 * ax,ay,(az) -- and, for continuity mode, every array gives arho -- the first
                                 * sph_pc_step reuses them as a^n instead of re-evaluating); output of sph_sync_state.
                                 * NULL -> 0 / not written. */
} sph_array;

typedef struct sph_stats {
    int32_t n_cells[3];         /* grid dimensions of the coarsest level (cells >= k h_max; n_cells[0] counts x sub-cells) */
    double cell_size[3];
    int64_t n_particles;        /* all arrays */
    int64_t pairs_density;      /* (i,j) pairs passing the exact predicate in the last density pass(es), self pairs included */
    int64_t pairs_accel;        /* same for the last acceleration pass(es) */
    int64_t candidates;         /* candidates streamed through the filter in the last density + acceleration passes */
    int64_t candidates_density, candidates_accel;   /* ... by pair passes that searched themselves (no record pool) */
    int64_t kernel_launches;    /* CUDA kernels launched by this context since sph_create */
    int64_t steps_done;         /* predictor-corrector steps since the last sph_nnps_build */
    int32_t variable_h;         /* 1 if h_min != h_max at the last build */
    float h_max;
    int32_t xsub;               /* x sub-cells per support radius of the current grid (n_cells[0] counts sub-cells) */
    int32_t used_rows;          /* 1 if the last acceleration pass replayed the candidate masks recorded by the search */
    int64_t nlist_rows_used, nlist_rows_capacity;   /* record pool occupancy after the last recording pass */
    int64_t nlist_fallback_warps;                   /* warps whose masks did not fit the pool in that pass (they search again) */
    int32_t n_levels;           /* h classes / level grids of the current build (1 when h is constant) */
    int64_t n_keys;             /* entries of the shared cell table (all levels x arrays) */
    int64_t candidates_search;  /* candidates streamed through the filter by the last search (one per sorted order) */
} sph_stats;

/* Per-kernel device timing (CUDA events on the context stream around every launch), for the roofline report. */
enum sph_kernel_id {
    SPH_K_PACK = 0,             /* caller SoA -> packed state + h_min/h_max                       */
    SPH_K_KEY = 1,              /* a1: cell key + histogram                                       */
    SPH_K_UPDATE = 2,           /* a8 + a1: predictor-corrector update fused with key + histogram */
    SPH_K_SCAN = 3,             /* a2: exclusive scan of the cell histogram                       */
    SPH_K_SCATTER = 4,          /* a2/a3: counting-sort scatter of every property into cell order */
    SPH_K_DENSITY = 5,          /* a4 + a5: summation density + EOS                               */
    SPH_K_ACCEL = 6,            /* a6 + a7: momentum (+ continuity) pair loop                     */
    SPH_K_OUTPUT = 7,           /* caller-order output gather                                     */
    SPH_K_NEIGHBORS = 8,        /* verification export                                            */
    SPH_K_ACCEL_LIST = 9,       /* a6 + a7 replayed over the candidate masks recorded by the search */
    SPH_K_SEARCH = 10,          /* neighbour search of one sorted order: tensor-core filter -> mask records */
    SPH_K_DENSITY_LIST = 11,    /* a4 + a5 replayed over the candidate masks recorded by the search */
    SPH_K_UPDATE_KICK = 12,     /* a8, eq.14 only (the launch that ends a sph_pc_step call): no drift, no key */
    SPH_K_SCAN_REDUCE = 13,     /* a2, tables of >= 1024 tiles: per-tile sums (SPH_K_SCAN is then the pass that applies them) */
    SPH_K_SCAN_TILES = 14,      /* a2, tables of >= 1024 tiles: exclusive scan of the tile sums (one block)     */
    SPH_K_COUNT = 16
};
typedef struct sph_profile {
    int64_t launches[SPH_K_COUNT];   /* launches recorded since sph_set_profiling(ctx, 1)         */
    double ms[SPH_K_COUNT];          /* summed device time of those launches                      */
    int64_t dropped;                 /* launches not recorded because the event pool was full     */
} sph_profile;

/* ---- lifetime ------------------------------------------------------------------------------- */

/* Creates a context for `n_arrays` (1..SPH_MAX_ARRAYS) particle arrays of at most capacity[a] particles.
 * cuda_stream: a cudaStream_t (e.g. torch.cuda.Stream.cuda_stream), NULL = the legacy default stream.
 * Allocates all workspace (about 190 B per particle of capacity + the cell tables + the record pool,
 * 768 B per particle of capacity by default, see sph_params.nlist_slots).  [sync] */
int sph_create(sph_ctx** out, const sph_params* params, const sph_domain* domain,
               int n_arrays, const int64_t* capacity, void* cuda_stream);
int sph_destroy(sph_ctx* ctx);                                                           /* [sync] */

/* Dest/source tables used by sph_pc_step (Listing 3; L528-534).  Each is an array of n_arrays
 * bitmasks over source arrays (bit b = array b); NULL keeps the default:
 *   density (summation mode): every array <- all arrays;
 *   accel:   dynamic arrays <- all arrays, fixed arrays <- none;
 *   arho (continuity mode):   dynamic <- all arrays, fixed <- dynamic arrays only. */
int sph_set_tables(sph_ctx* ctx, const uint32_t* density_src, const uint32_t* accel_src, const uint32_t* arho_src);

/* ---- the four calls of the path --------------------------------------------------------------- */

/* sph_nnps_build(pos, h, domain, periodic) -- Sec.2.2 (L158-170): loads the caller's arrays (positions and
 * h define the search; u,v,w,m,rho,p are carried along into cell order), computes h_max, sizes the cell
 * grid (cell >= k*h_max, L158-160), computes cell keys, counting-sorts all arrays into ONE grid (key =
 * cell * n_arrays + array), builds cell-start offsets and gathers every property into cell order.
 * Replaces any previous state of the context.  [sync] (reads h_max back to size the grid) */
int sph_nnps_build(sph_ctx* ctx, int n_arrays, const sph_array* arrays);

/* Summation density, eq.3 (L112): rho_i = sum_{b in source_mask} sum_{j in N_b(i)} m_j W(r_ij, h_ij) for
 * every particle i of array `dest`, self pair included; then the EOS (eq.6) on that array.  Updates the
 * context's rho/p of `dest` and, if non-NULL, writes rho_out / p_out (n_dest reals, caller order, `mem`). */
int sph_summation_density(sph_ctx* ctx, int dest, uint32_t source_mask, sph_real* rho_out, sph_real* p_out, int mem);

/* WCSPH acceleration, eq.8-9 (L128-132) + artificial viscosity + optional continuity RHS eq.7 (L126):
 *   a_i = g - sum_b sum_j m_j (p_i/rho_i^2 + p_j/rho_j^2 + Pi_ij) grad_i W_ij,   arho_i = sum m_j v_ij . grad_i W_ij
 * from the context's current rho,p (as loaded by sph_nnps_build or computed by sph_summation_density).
 * ax,ay,az (az may be NULL when dim == 2) and arho (NULL: not computed) receive n_dest floats, caller order. */
int sph_wcsph_accel(sph_ctx* ctx, int dest, uint32_t source_mask,
                    sph_real* ax, sph_real* ay, sph_real* az, sph_real* arho, int mem);

/* n_steps time steps on the context's state.  sph_params.integrator == SPH_INTEGRATOR_EULER: forward Euler
 * (see enum sph_integrator), one evaluation per step.  Default: predictor-corrector, eqs. 12-14 (L148-152),
 * DESIGN.md R10/R11:
 *   [a^0 = F(x^0,u^0) on the first call after a build]
 *   u += dt/2 a ; x += dt u (+ periodic wrap, L443) ; NNPS rebuilt (L443) ; [rho = eq.3] ; EOS ; a = F ; u += dt/2 a
 * density_mode selects eq.3 or the integrated eq.7 (rho stepped like u, on every array).
 * Fixed arrays keep x,u.  No host synchronisation inside. */
int sph_pc_step(sph_ctx* ctx, double dt, int n_steps, int density_mode);

/* ---- state out, verification, diagnostics ------------------------------------------------------ */

/* Writes the context's current state of array `array` into the non-NULL pointers of *out
 * (x,y,z,u,v,w,rho,p,ax,ay,az,arho; h and m never change) in the caller's original particle order.  out->n must equal
 * the array's size.  Asynchronous for SPH_MEM_DEVICE; [sync] for SPH_MEM_HOST. */
int sph_sync_state(sph_ctx* ctx, int array, const sph_array* out);

/* Last accelerations of array `array` (ax,ay,az,arho; any may be NULL), caller order. */
int sph_get_accel(sph_ctx* ctx, int array, sph_real* ax, sph_real* ay, sph_real* az, sph_real* arho, int mem);

/* Neighbour lists N_src(i) of every particle i of array `dest` as CSR in ORIGINAL indices of array `src`,
 * each row sorted ascending: offsets[n_dest+1], indices[total].  Pass indices == NULL (or too small a cap)
 * to get *total only.  Used for the bit-exact set parity.  Host pointers when mem == SPH_MEM_HOST.  [sync] */
int sph_nnps_get_neighbors(sph_ctx* ctx, int dest, int src, int64_t* offsets, int32_t* indices,
                           int64_t cap, int64_t* total, int mem);

/* enable != 0: record a CUDA event pair around every kernel launch from now on (clears earlier records);
 * 0: stop.  Off by default (the events add a few microseconds per launch). */
int sph_set_profiling(sph_ctx* ctx, int enable);
int sph_get_profile(sph_ctx* ctx, sph_profile* out);                                     /* [sync] */
const char* sph_kernel_name(int kernel_id);

int sph_get_stats(sph_ctx* ctx, sph_stats* out);                                         /* [sync] */
int sph_synchronize(sph_ctx* ctx);   /* [sync] waits for the stream and reports pending device-side errors */

/* Diagnostic, not a step of the path: sustained FP32 fused-multiply-add rate of this GPU, scalar (packed == 0,
 * FFMA) or packed (packed != 0, FFMA2), over `iters` iterations of 16 independent accumulators per thread on
 * 8 blocks of 256 threads per SM.  *tflops counts 2 flop per lane FMA; *ms (nullable) is the best of 3 timed
 * launches.  It is the measured denominator of the pair kernels' ALU roofline.  [sync] */
int sph_fp32_probe(sph_ctx* ctx, int packed, int iters, double* tflops, double* ms);

/* Diagnostic, not a step of the path: the size of the candidate set of the PAPER's cell-list search on the current
 * state -- sum over all particles of the population of the 3^d cells of size >= k*h_max around them (L158, one
 * uniform grid sized by h_max).  It is the work unit the roofline report charges a searching pass with, whatever
 * this library really tests (sph_stats.candidates*).  Positions in the cell-sorted mirror are used.  [sync] */
int sph_stencil_candidates(sph_ctx* ctx, int64_t* out);

/* Allocation-free cell offsets (Sec.2.2: the start of every cell's run in the cell-sorted order = the
 * exclusive prefix sum of the per-cell particle counts), for callers that may not call cudaMalloc (code under CUDA
 * graph capture, tight serving loops, harnesses that forbid it).  It needs no context: it is the single-pass
 * look-back scan of the sort (k_scan) with its look-back table in a file-scope device array of the library instead
 * of in memory the context allocates.
 *   d_counts   DEVICE pointer, n uint32 (read only, caller-owned)
 *   d_offsets  DEVICE pointer, n + 1 uint32 (written; [n] = the total, which must fit 32 bits), caller-owned,
 *              must not overlap d_counts
 *   n          0 <= n <= SPH_STATIC_SCAN_MAX_N; n == 0 writes d_offsets[0] = 0
 *   stream     a cudaStream_t of the CURRENT device (NULL = the default stream); the call is asynchronous on it
 * The call issues one cudaMemsetAsync and one kernel and calls no cudaMalloc / cudaFree / allocating routine.  The
 * first call on each device looks up the device address of the array (cudaGetSymbolAddress): make that first call
 * (n = 0 will do) outside stream capture.  The array (SPH_STATIC_SCAN_BYTES, about 128 KiB) is held by every GPU
 * that loads the library until the process exits, and is SHARED by all calls on that GPU: each call clears the
 * part it uses, so calls in stream order are independent of one another, but two calls that overlap on the GPU
 * (different streams, no dependency between them) race on it and give wrong offsets.
 * Errors: SPH_ERR_NULL (a pointer is NULL and n > 0, or d_offsets is NULL), SPH_ERR_BAD_ARG (n < 0),
 * SPH_ERR_CAPACITY (n > SPH_STATIC_SCAN_MAX_N), SPH_ERR_CUDA; sph_static_last_error() gives the message of the
 * calling thread's last failure (there is no context to hold it). */
#define SPH_STATIC_SCAN_MAX_N  67108864LL                           /* 2^26 counts per call */
#define SPH_STATIC_SCAN_BYTES  (256 + 8 * (SPH_STATIC_SCAN_MAX_N / 4096))   /* header + one word per 4096-count tile */
int sph_cell_offsets_static(const uint32_t* d_counts, int64_t n, uint32_t* d_offsets, void* stream);
const char* sph_static_last_error(void);

const char* sph_strerror(int code);
const char* sph_last_error(const sph_ctx* ctx);
int sph_abi_version(void);
int sph_real_size(void);              /* sizeof(sph_real) of the loaded library: 4 or 8 */

#ifdef __cplusplus
}
#endif
#endif /* SPH_B200_H */
