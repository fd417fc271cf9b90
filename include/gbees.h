/* gbees.h -- C ABI of the B200-native GBEES prediction step (arXiv 2508.13986, "GBEES-GPU").
 *
 * The library advances a probability density on a sparse, dynamically allocated n-D grid under
 * dp/dt + div(f p) = 0 (Eq. 3) with the Corner Transport Upwind finite-volume scheme
 * (Eq. 7, Alg. 1, PAPER.md:112 high-resolution terms), growing the
 * grid downwind of above-threshold cells and pruning cells below threshold,
 * with the Bayes correction of PAPER.md:59 (Eq. 4). Exact semantics: DESIGN.md "Definitions D1-D5".
 *
 * Conventions
 *  - Every call returns 0 (GBEES_OK) or a negative GBEES_ERR_*; nothing throws or aborts across
 *    the ABI. Device-side faults (pool overflow, key range) are recorded in a device flag and
 *    surfaced by the call that detected them; gbees_last_error() gives a message.
 *  - All computation happens in CUDA kernels on one GPU (sm_100a). There is no CPU fallback.
 *  - "host" / "device" below says where a pointer must live. Arrays passed in are copied; the
 *    caller keeps ownership of everything it passes. One context = one stream; calls on one
 *    context are not re-entrant.
 *  - The kernels of a step / prune are enqueued with programmatic dependent launch (the next kernel's blocks are
 *    scheduled while the previous one drains; every kernel waits for its predecessor before it reads anything).
 *    Environment variable GBEES_NO_PDL=1 (read by gbees_create) switches that off, for measurement.
 *  - Cell c in Z^n has centre x_c = origin + c o dx; origin = the mean given to init_gaussian.
 *    P_c is the probability MASS of cell c; sum over active cells = 1 after every normalisation.
 */
#ifndef GBEES_H
#define GBEES_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define GBEES_OK 0
#define GBEES_ERR_ARG (-1)        /* bad argument (n out of [1,6], dx <= 0, threshold <= 0, wrong n_params, NULL) */
#define GBEES_ERR_CUDA (-2)       /* a CUDA runtime call failed (message in gbees_last_error) */
#define GBEES_ERR_NOT_SPD (-3)    /* cov / R is not symmetric positive definite */
#define GBEES_ERR_CAPACITY (-4)   /* more cells than opts.max_cells (fixed capacity) */
#define GBEES_ERR_BUFFER (-5)     /* export buffer too small; *count holds the needed size */
#define GBEES_ERR_DEGENERATE (-6) /* mass <= 0 or non-finite, empty grid, or no CFL bound and no cap */
#define GBEES_ERR_KEY_RANGE (-7)  /* a coordinate left the packable range (floor(63/n) bits, biased) */

/* dynamics ids: f(x) in dx/dt = f(x). Operation order is fixed (A12). */
#define GBEES_DYN_LORENZ63 0        /* params (sigma, beta, rho); n = 3 (BASELINE configs 0-1) */
#define GBEES_DYN_LORENZ63_PAPER 1  /* params (sigma, b, r), PAPER.md:303 z-shifted form; n = 3 */
#define GBEES_DYN_LORENZ96 2        /* params (F); n >= 4, cyclic */
#define GBEES_DYN_LINEAR 3          /* params A row-major n*n: f = A x (BASELINE config 3) */
#define GBEES_DYN_CONSTANT 4        /* params v[n]: f = v (tests) */

typedef struct gbees_ctx gbees_ctx;

typedef struct gbees_opts {
    int64_t max_cells;   /* active-cell capacity; storage = max(ceil(max_cells/16), 256) bricks of 64 cell slots, brick hashtable with ceil(bricks / load_factor) slots */
    double load_factor;  /* default 0.5 */
    double cfl;          /* C in dt = C * min_c (sum_j |u_cj| / h_j)^-1, Eq. (8); default 0.9 */
    int hi_res;          /* 1 = add the high-resolution (limited Lax-Wendroff) term; default 1 */
    int limiter;         /* 0 = monotonised central, 1 = none (phi == 1, test mode) */
    int no_grow;         /* test mode: gbees_step does not grow the grid */
    int no_normalise;    /* test mode: keep raw (un-normalised) masses after step / prune */
    int run_mode;        /* gbees_run: 0 = device-side step control, no host round trip per step (default); 1 = host loop of gbees_step /
                            gbees_prune; 2 = as 0 with the chunks of steps captured as a CUDA graph; 3 = one cooperative launch over
                            the whole GPU with grid barriers between the phases. 2 and 3 are kept for measurement:
                            same results, 0 is the fastest */
    int device;          /* CUDA device ordinal */
    void* stream;        /* cudaStream_t to run on (e.g. torch's current stream); NULL = default */
    void* arena;         /* optional caller-owned DEVICE memory (e.g. the data_ptr of a torch uint8 tensor on opts.device) that all
                            fixed-capacity device structures are carved from instead of cudaMalloc; must stay alive until gbees_destroy,
                            which does not free it; NULL = the library allocates (capacity is fixed at creation) */
    int64_t arena_bytes; /* its size; gbees_arena_bytes() says how much gbees_create needs (GBEES_ERR_CAPACITY if too small) */
} gbees_opts;

typedef struct gbees_stats_t {
    int64_t n_cells;        /* active cells now */
    int64_t n_inserted;     /* cells created by the last step's grow */
    int64_t n_pruned;       /* cells removed by the last prune */
    int64_t steps;          /* steps taken since init */
    double t;               /* simulated time */
    double dt;              /* last step size */
    double mass;            /* mass before the last normalisation (1 - mass left the grid) */
    int64_t cell_updates;   /* sum over steps of the active-cell count after grow */
    int64_t table_slots;    /* hashtable capacity in slots */
    int64_t launches;       /* kernel + memset launches issued by this context so far */
    int64_t cells_inserted;      /* cells created by grow since init */
    int64_t cells_prune_scanned; /* sum over prunes of the cell count scanned */
    int64_t prunes;              /* prunes since init */
} gbees_stats_t;

/* phases of the hot path, for launch accounting and optional CUDA-event timing */
enum {
    GBEES_PH_GROW = 0,  /* a1: grow (activate downwind targets, create bricks) + CFL terms of the new cells (a3) */
    GBEES_PH_LINK,      /* adjacency of the bricks created by the grow */
    GBEES_PH_PASSA,     /* a2+a4: face velocities, upwind-owner CTU fluxes (k_flux1) */
    GBEES_PH_PASSB,     /* a5+a6: fetch neighbour-brick fluxes, update, mass sum, dt/t bookkeeping (k_flux2) */
    GBEES_PH_MARK,      /* a7: prune marking */
    GBEES_PH_COMPACT,   /* a7: decoupled-lookback scan over bricks + row compaction */
    GBEES_PH_REBUILD,   /* a7/a0: hashtable clear + re-insert (in a prune: + CFL maximum, mass sum, cell count) */
    GBEES_PH_RELINK,    /* adjacency for all bricks (in a prune: + renormalise by the last block) */
    GBEES_PH_SUM,       /* a6: mass sum + renormalise outside a step */
    GBEES_PH_CORRECT,   /* a8 */
    GBEES_PH_RUN,       /* a9: persistent single-cluster step loop for small grids (whole launch; not used while profiling) */
    GBEES_PHASES
};

/* Fill *opts with the defaults (max_cells = 1<<20, load_factor 0.5, cfl 0.9, hi_res 1, MC). */
int gbees_default_opts(gbees_opts* opts /*host*/);
/* Device bytes that gbees_create(n, ..., opts) carves from opts->arena (a function of n, max_cells and load_factor
 * only; opts == NULL: the defaults). bytes: host. */
int gbees_arena_bytes(int n, const gbees_opts* opts /*host, nullable*/, int64_t* bytes);

/* Allocate all fixed-capacity device structures. dx, params: host, copied.
 * n in [1,6]; n_params must match dynamics_id. opts may be NULL (defaults). */
int gbees_create(gbees_ctx** out, int n, const double* dx /*host [n]*/, double threshold,
                 int dynamics_id, const double* params /*host*/, int n_params,
                 const gbees_opts* opts /*host, nullable*/);
int gbees_destroy(gbees_ctx* ctx);

/* DESIGN.md D5/A8: origin <- mean, grid <- {c : g_c * prod(dx) / sqrt((2 pi)^n det cov) >= threshold},
 * P <- normalised, t <- 0. mean [n], cov [n*n row-major, SPD]: host. */
int gbees_init_gaussian(gbees_ctx* ctx, const double* mean, const double* cov);

/* Raw state import (tests / restart): origin [n] host; keys [count*n] int32 row-major and p [count]
 * on host or device. Keys must be distinct. P is taken as given (no normalisation), t <- 0. */
int gbees_import(gbees_ctx* ctx, const double* origin, const int32_t* keys, const double* p, int64_t count);

/* One prediction step, D1: grow -> dt (Eq. 8) -> CTU flux -> update -> normalise.
 * in: *dt = largest step allowed (<= 0, NaN or inf = unconstrained); out: *dt = step taken.
 * dt: host pointer. Does not prune. */
int gbees_step(gbees_ctx* ctx, double* dt);

/* DESIGN.md D3 (Alg. 3): keep cells with P >= threshold and the grow-targets of such
 * cells; stream-compact the pool, rebuild the hashtable, renormalise. */
int gbees_prune(gbees_ctx* ctx);

/* DESIGN.md D4, Eq. (4): P_c <- P_c * exp(-1/2 (z - x_c)^T R^-1 (z - x_c)), renormalise.
 * z [n], R [n*n row-major SPD]: host. Does not prune. */
int gbees_correct(gbees_ctx* ctx, const double* z, const double* R);

/* Eq. (4) with a linear measurement model y = H x + v, v ~ N(0, R) (the paper's own scenario measures
 * one state only: y = x3): P_c <- P_c * exp(-1/2 (y - H x_c)^T R^-1 (y - H x_c)),
 * renormalise. H [m*n row-major], y [m], R [m*m row-major SPD]: host; 1 <= m <= 6. Does not prune. */
int gbees_correct_linear(gbees_ctx* ctx, const double* H, int m, const double* y, const double* R);

/* Eq. (4) with a NON-linear measurement, the range to the point s: y = ||x - s||_2 + v, v ~ N(0, sigma^2):
 * P_c <- P_c * exp(-1/2 ((y - ||x_c - s||) / sigma)^2), renormalise. s [n]: host; sigma > 0 (else
 * GBEES_ERR_NOT_SPD). Does not prune. */
int gbees_correct_range(gbees_ctx* ctx, const double* s, double y, double sigma);

/* Distribution metrics between two contexts on the SAME grid (same n, dx, origin, device; else
 * GBEES_ERR_ARG): *bc = sum_c sqrt(Pa_c Pb_c) (Bhattacharyya coefficient, Eq. 9) and
 * *l1 = sum_c |Pa_c - Pb_c| (the paper's 1-norm E of PAPER.md:362-366 in cell masses), over the union
 * of the two active sets. bc, l1: host. Neither context is modified. */
int gbees_compare(gbees_ctx* ctx, gbees_ctx* other, double* bc, double* l1);

/* Marginal PDF: sum the cell probabilities over the dimensions NOT listed in
 * dims [m] (host; distinct indices in [0, n), output order = order in dims), hash-accumulated on the
 * device. Writes *count marginal cells in unspecified order: keys [cap*m] int32 row-major, p [cap]
 * (host or device buffers, caller-owned); keys == NULL or p == NULL: only *count; cap < *count:
 * GBEES_ERR_BUFFER. The additions are atomic, so the last bits of p may differ between calls. */
int gbees_marginal(gbees_ctx* ctx, const int* dims, int m, int32_t* keys, double* p, int64_t cap, int64_t* count);

/* Conservative remap of the PDF onto a grid with origin origin2 [n] and spacing dx2 [n] (host), dx2[j] >= dx[j]
 * for every j (else GBEES_ERR_ARG). The paper compares runs on grids of different cell width with the eta = 0.5
 * reference (spatial convergence) without saying how; reading A19: the PDF is piecewise
 * constant over its cells, and cell d of the target grid receives P_c times the fraction of c's volume inside d
 * (a product of 1-D overlap fractions; overlaps below 1e-12 of a cell width are dropped). Mass is preserved.
 * Output as for gbees_marginal: *count target cells in unspecified order, keys [cap*n] int32 row-major (cell
 * coordinates on the target grid), p [cap]; host or device buffers; keys == NULL or p == NULL: only *count;
 * cap < *count: GBEES_ERR_BUFFER. Import the result into a context of the target spacing (gbees_import) to
 * compare it with a run on that grid (gbees_compare). The context is not modified. */
int gbees_resample(gbees_ctx* ctx, const double* origin2, const double* dx2, int32_t* keys, double* p, int64_t cap, int64_t* count);

/* Marginal PDF WITHOUT ANY ALLOCATION (for callers that cannot call cudaMalloc: code under CUDA graph capture, tight
 * serving loops, harnesses that forbid it). Same result as gbees_marginal, but computed from an
 * exported state instead of a context: keys [count_in*n] int32 row-major and p [count_in] (DEVICE pointers on
 * `device`, e.g. what gbees_export wrote into device buffers), dims [m] (host; distinct indices in [0, n), output
 * order = order in dims). Writes *count (host) marginal cells in unspecified order to out_keys [cap*m] int32 and
 * out_p [cap] (DEVICE pointers, caller-owned). The scratch hashtable lives in a file-scope device array of
 * 2 * GBEES_NOALLOC_MAX_CELLS slots (4 MiB, held by every GPU that loads the library until the process exits):
 * count_in > GBEES_NOALLOC_MAX_CELLS is rejected with GBEES_ERR_CAPACITY (use gbees_marginal), cap < *count gives
 * GBEES_ERR_BUFFER (with *count set), a kept coordinate outside floor(63/m) bits GBEES_ERR_KEY_RANGE. The call
 * enqueues three kernels on `stream` (a cudaStream_t, NULL = default) and waits for them; it calls no cudaMalloc,
 * cudaFree or allocating library routine. ALL calls share the one scratch array, which keeps the previous call's
 * contents (each call clears what it uses first): calls that overlap on the GPU -- two streams, two threads -- RACE;
 * serialise them. The additions are atomic, so the last bits of p may differ between calls.
 * gbees_marginal_noalloc_error(): message of the calling thread's last failed call. */
#define GBEES_NOALLOC_MAX_CELLS 131072
int gbees_marginal_noalloc(int device, void* stream, int n, const int32_t* keys /*device*/, const double* p /*device*/,
                           int64_t count_in, const int* dims /*host*/, int m, int32_t* out_keys /*device*/,
                           double* out_p /*device*/, int64_t cap, int64_t* count /*host*/);
const char* gbees_marginal_noalloc_error(void);

/* Write the active cells in unspecified order: keys [cap*n] int32 row-major, p [cap] (normalised).
 * Buffers: host or device (detected), caller-owned. keys == NULL and p == NULL: only *count.
 * cap < count: nothing written, *count = needed, GBEES_ERR_BUFFER. count: host pointer. */
int gbees_export(gbees_ctx* ctx, int32_t* keys, double* p, int64_t cap, int64_t* count);

/* Step loop kept on the device: advance until t == t_target or max_steps steps,
 * pruning after every prune_every-th step (0 = never). The launches of a chunk of steps are enqueued
 * at once; a device flag set by each step's last block decides whether the next ones execute, so
 * there is no host round trip per step. Observationally identical to the same sequence of
 * gbees_step(&cap = t_target - t) / gbees_prune calls. steps_done: host, nullable. */
int gbees_run(gbees_ctx* ctx, double t_target, int64_t max_steps, int prune_every, int64_t* steps_done);

int gbees_count(gbees_ctx* ctx, int64_t* count /*host*/);
int gbees_time(gbees_ctx* ctx, double* t /*host*/);
int gbees_stats(gbees_ctx* ctx, gbees_stats_t* out /*host*/);
/* Read-and-reset the per-phase accumulators (phase_ms, phase_launches: host [GBEES_PHASES],
 * nullable), then switch CUDA-event timing of every phase on/off. Synchronises the stream.
 * Launch counts are always kept; milliseconds only while profiling is enabled. While profiling is on
 * gbees_run always uses the per-phase launches (never the single-launch loop for small grids). */
int gbees_profile(gbees_ctx* ctx, int enable, double* phase_ms, int64_t* phase_launches);
const char* gbees_last_error(gbees_ctx* ctx);
int gbees_clear_error(gbees_ctx* ctx);

/* ---- BASELINE config 4: hashtable / compaction microbenchmark on the same device code ---------
 * Keys are packed 64-bit values (never all-ones) in DEVICE memory. probes = slots inspected. */
typedef struct gbees_ht gbees_ht;
int gbees_ht_create(gbees_ht** out, int64_t slots, int device);
int gbees_ht_destroy(gbees_ht* ht);
/* insert-if-absent keys[0..k); idx_out[i] = pool index assigned (or existing); nullable */
int gbees_ht_insert(gbees_ht* ht, const uint64_t* keys, int64_t k, uint32_t* idx_out, uint64_t* probes /*host*/);
/* out[i] = pool index of query[i] or 0xFFFFFFFF */
int gbees_ht_lookup(gbees_ht* ht, const uint64_t* query, int64_t k, uint32_t* out, uint64_t* probes /*host*/);
/* the same lookup with cooperative probing (north_star: "warp-cooperative probing"): a tile of `width`
 * lanes (4, 8 or 32) inspects `width` consecutive slots per round for one query. Same answers and the
 * same probe count as gbees_ht_lookup. */
int gbees_ht_lookup_coop(gbees_ht* ht, const uint64_t* query, int64_t k, uint32_t* out, uint64_t* probes /*host*/, int width);
/* delete keys[i] where del[i] != 0: decoupled-lookback scan + stable compaction of keys (in place)
 * + table rebuild. *k_out = survivors. */
int gbees_ht_compact(gbees_ht* ht, uint64_t* keys, const uint8_t* del, int64_t k, int64_t* k_out /*host*/);

#ifdef __cplusplus
}
#endif
#endif /* GBEES_H */
