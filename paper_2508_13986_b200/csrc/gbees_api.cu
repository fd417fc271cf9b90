// Host side of the C ABI in include/gbees.h: context, launches, error handling.
// All arithmetic of the method runs in the kernels of gbees_kernels.cuh; the host only computes
// the launch-invariant inputs of init_gaussian / correct (an n x n Cholesky inverse, n <= 6).
#include <cmath>
#include <cstdio>
#include <cstring>
#include <string>
#include <utility>
#include <vector>

#include "../../include/gbees.h"
#include "gbees_kernels.cuh"

using namespace gbees;

// ------------------------------------------------------------------------------------------------
// __global__ wrappers (one per phase; Params by value in constant bank)
// ------------------------------------------------------------------------------------------------
__global__ void k_begin(DevState* st, double dt_cap) {
    st->N_before_grow = st->N;
    st->dt_cap = dt_cap;
}
template <int NDIM, int DYN>
__global__ void __launch_bounds__(TPB) k_grow(const __grid_constant__ Params p, const __grid_constant__ Pool pool, DevState* st) {
    phase_grow<NDIM, DYN>(p, pool, st);
}
template <int NDIM, int DYN, bool ALL>
__global__ void __launch_bounds__(TPB) k_link(const __grid_constant__ Params p, const __grid_constant__ Pool pool, DevState* st) {
    phase_link<NDIM, DYN, ALL>(p, pool, st);
}
template <int NDIM, int DYN>
__global__ void __launch_bounds__(PassACfg<NDIM>::BLK) k_passA(const __grid_constant__ Params p, const __grid_constant__ Pool pool, DevState* st) {
    phase_passA<NDIM, DYN>(p, pool, st);
}
template <int NDIM>
__global__ void __launch_bounds__(TPB) k_passB(const __grid_constant__ Params p, const __grid_constant__ Pool pool, DevState* st) {
    phase_passB<NDIM>(p, pool, st);
}
__global__ void __launch_bounds__(TPB) k_sum(const __grid_constant__ Params p, const __grid_constant__ Pool pool, DevState* st) {
    phase_sum(p, pool, st);
}
// mode: 0 = after a step, 1 = renormalise only (init / correct / prune), 2 = sum only (import)
__global__ void __launch_bounds__(TPB) k_finish(const __grid_constant__ Params p, const __grid_constant__ Pool pool, DevState* st,
                                                unsigned nparts, int mode) {
    Params q = p;
    if (mode == 2) q.normalise = 0;
    finish_sum(q, pool, st, nparts, mode == 0);
}
template <int NDIM, int DYN>
__global__ void __launch_bounds__(TPB) k_mark(const __grid_constant__ Params p, const __grid_constant__ Pool pool, DevState* st) {
    phase_mark<NDIM, DYN>(p, pool, st);
}
__global__ void __launch_bounds__(TPB) k_compact(const __grid_constant__ Params p, const __grid_constant__ Pool pool, DevState* st) {
    phase_compact(p, pool, st);
}
__global__ void k_after_compact(const __grid_constant__ Params p, DevState* st) {
    st->prune_scanned += st->N;
    st->prunes += 1;
    st->N_before_grow = st->N;          // old row count, read by the adjacency remap
    st->N = st->N_after_prune;
    st->slots = table_slots_for(p, st->N);
    st->smax_bits = 0ull;
    st->tile_counter = 0u;
}
__global__ void k_set_slots(const __grid_constant__ Params p, DevState* st) {
    st->slots = table_slots_for(p, min(st->N, p.cap));
    st->smax_bits = 0ull;
}
__global__ void __launch_bounds__(TPB) k_clear_table(const __grid_constant__ Pool pool, const DevState* st) {
    phase_clear_table(pool, st);
}
// prune: translate the adjacency through newidx (into nbr2) and clear the resized table
__global__ void __launch_bounds__(TPB) k_remap_clear(const __grid_constant__ Params p, const __grid_constant__ Pool pool, const DevState* st) {
    phase_remap(p, pool, st->N_before_grow, 2 * p.n);
    phase_clear_table(pool, st);
}
__global__ void __launch_bounds__(TPB) k_rebuild(const __grid_constant__ Params p, const __grid_constant__ Pool pool, DevState* st) {
    phase_rebuild(p, pool, st);
}
// prune tail: re-insert all keys, recompute the CFL maximum, sum the masses
template <int NDIM, int DYN>
__global__ void __launch_bounds__(TPB) k_rebuild_smax_sum(const __grid_constant__ Params p, const __grid_constant__ Pool pool, DevState* st) {
    phase_rebuild(p, pool, st);
    phase_smax<NDIM, DYN>(p, pool, st);
    phase_sum(p, pool, st);
}
template <int NDIM>
__global__ void __launch_bounds__(TPB) k_init_gaussian(const __grid_constant__ Params p, const __grid_constant__ Pool pool, DevState* st,
                                                       const __grid_constant__ GaussArgs g) {
    phase_init_gaussian<NDIM>(p, pool, st, g);
}
template <int NDIM>
__global__ void __launch_bounds__(TPB) k_correct(const __grid_constant__ Params p, const __grid_constant__ Pool pool, DevState* st,
                                                 const __grid_constant__ GaussArgs g) {
    phase_correct<NDIM>(p, pool, st, g);
}
template <int NDIM>
__global__ void __launch_bounds__(TPB) k_export(const __grid_constant__ Params p, const __grid_constant__ Pool pool, const DevState* st,
                                                int32_t* keys, double* out) {
    phase_export<NDIM>(p, pool, st, keys, out);
}
template <int NDIM>
__global__ void __launch_bounds__(TPB) k_import(const __grid_constant__ Params p, const __grid_constant__ Pool pool, DevState* st,
                                                const int32_t* keys, const double* vals, uint32_t count) {
    phase_import<NDIM>(p, pool, st, keys, vals, count);
}

template <int NDIM, int DYN>
__global__ void __launch_bounds__(TPB) k_run(const __grid_constant__ Params p, const __grid_constant__ Pool pool, DevState* st,
                                             const __grid_constant__ RunArgs a) {
    phase_run<NDIM, DYN>(p, pool, st, a);
}

// ------------------------------------------------------------------------------------------------
// context
// ------------------------------------------------------------------------------------------------
struct gbees_ctx {
    Params p{};
    Pool pool{};
    DevState* d_st = nullptr;
    DevState* h_st = nullptr;  // pinned mirror
    cudaStream_t stream = nullptr;
    int device = 0;
    int sms = 148;
    unsigned grid = 148 * 8;
    unsigned grid_passA = 148 * 8;
    unsigned ntiles_max = 0;
    int sticky = 0;
    int no_grow = 0;
    int run_mode = 0;            // 0 = persistent cooperative kernel, 1 = host loop over step/prune
    int run_blocks_per_sm = 0;
    int64_t n_inserted = 0, n_pruned = 0;
    std::string err;
    void* allocs[24] = {nullptr};
    int nallocs = 0;
    // launch accounting + optional per-phase CUDA-event timing (gbees_profile)
    int64_t launches = 0;
    int profile = 0;
    std::vector<cudaEvent_t> ev_free;
    std::vector<std::pair<int, std::pair<cudaEvent_t, cudaEvent_t>>> ev_open;
    double phase_ms[GBEES_PHASES] = {0};
    double run_phase_ms[GBEES_PHASES] = {0};   // breakdown inside the persistent kernel (device timer)
    int run_ns_dirty = 0;
    int64_t phase_launches[GBEES_PHASES] = {0};
};

namespace {

int fail(gbees_ctx* c, int code, const std::string& msg) {
    if (c) { c->err = msg; c->sticky = code; }
    return code;
}
#define CU(call)                                                                                      \
    do {                                                                                              \
        cudaError_t e_ = (call);                                                                      \
        if (e_ != cudaSuccess)                                                                        \
            return fail(c, GBEES_ERR_CUDA, std::string(#call) + ": " + cudaGetErrorString(e_));       \
    } while (0)

// run `body` (kernel launches) as one accounted phase; with profiling on, bracket it with events
template <typename F>
void phase(gbees_ctx* c, int ph, int nlaunch, F&& body) {
    c->launches += nlaunch;
    c->phase_launches[ph] += nlaunch;
    if (!c->profile) { body(); return; }
    cudaEvent_t a, b;
    auto get = [&](cudaEvent_t* e) {
        if (c->ev_free.empty()) cudaEventCreate(e);
        else { *e = c->ev_free.back(); c->ev_free.pop_back(); }
    };
    get(&a); get(&b);
    cudaEventRecord(a, c->stream);
    body();
    cudaEventRecord(b, c->stream);
    c->ev_open.push_back({ph, {a, b}});
}
void drain_events(gbees_ctx* c) {   // call after a stream sync
    for (auto& e : c->ev_open) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, e.second.first, e.second.second) == cudaSuccess) c->phase_ms[e.first] += ms;
        c->ev_free.push_back(e.second.first);
        c->ev_free.push_back(e.second.second);
    }
    c->ev_open.clear();
}

template <int V> struct IC { static constexpr int value = V; };

// call f(IC<NDIM>, IC<DYN>) for the context's (n, dynamics) pair; only valid pairs are instantiated
template <typename F>
int dispatch(const gbees_ctx* c, F&& f) {
    const int n = c->p.n, d = c->p.dyn;
#define GB_CASE(N_, D_) if (n == N_ && d == D_) return f(IC<N_>{}, IC<D_>{});
    GB_CASE(3, 0) GB_CASE(3, 1)
    GB_CASE(4, 2) GB_CASE(5, 2) GB_CASE(6, 2)
    GB_CASE(1, 3) GB_CASE(2, 3) GB_CASE(3, 3) GB_CASE(4, 3) GB_CASE(5, 3) GB_CASE(6, 3)
    GB_CASE(1, 4) GB_CASE(2, 4) GB_CASE(3, 4) GB_CASE(4, 4) GB_CASE(5, 4) GB_CASE(6, 4)
#undef GB_CASE
    return GBEES_ERR_ARG;
}
template <typename F>
int dispatch_n(const gbees_ctx* c, F&& f) {
    switch (c->p.n) {
        case 1: return f(IC<1>{}); case 2: return f(IC<2>{}); case 3: return f(IC<3>{});
        case 4: return f(IC<4>{}); case 5: return f(IC<5>{}); case 6: return f(IC<6>{});
    }
    return GBEES_ERR_ARG;
}

// Cholesky inverse of an SPD n x n matrix (host; n <= 6) and its determinant
bool spd_inverse(int n, const double* A, double* inv, double* det) {
    double L[MAXN][MAXN] = {{0}}, Li[MAXN][MAXN] = {{0}};
    for (int i = 0; i < n; ++i)
        for (int j = 0; j <= i; ++j) {
            if (std::fabs(A[i * n + j] - A[j * n + i]) > 1e-12 * (std::fabs(A[i * n + j]) + std::fabs(A[j * n + i]))) return false;
            double s = A[i * n + j];
            for (int k = 0; k < j; ++k) s -= L[i][k] * L[j][k];
            if (i == j) { if (!(s > 0.0)) return false; L[i][i] = std::sqrt(s); }
            else L[i][j] = s / L[j][j];
        }
    for (int i = 0; i < n; ++i) {
        Li[i][i] = 1.0 / L[i][i];
        for (int j = 0; j < i; ++j) {
            double s = 0.0;
            for (int k = j; k < i; ++k) s -= L[i][k] * Li[k][j];
            Li[i][j] = s / L[i][i];
        }
    }
    double d = 1.0;
    for (int i = 0; i < n; ++i) d *= L[i][i] * L[i][i];
    *det = d;
    for (int i = 0; i < n; ++i)
        for (int j = 0; j < n; ++j) {
            double s = 0.0;
            for (int k = (i > j ? i : j); k < n; ++k) s += Li[k][i] * Li[k][j];
            inv[i * n + j] = s;
        }
    return true;
}

// copy the device state to the pinned mirror, wait, translate device error bits
int sync_state(gbees_ctx* c) {
    CU(cudaMemcpyAsync(c->h_st, c->d_st, sizeof(DevState), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    if (c->profile) drain_events(c);
    // persistent loop: fold the device-timer phase breakdown into the accumulators
    for (int k = 0; k < GBEES_PH_RUN; ++k)
        if (c->h_st->phase_ns[k]) {
            c->run_phase_ms[k] += 1e-6 * (double)c->h_st->phase_ns[k];
            c->h_st->phase_ns[k] = 0;
            c->run_ns_dirty = 1;
        }
    if (c->run_ns_dirty) {
        cudaMemsetAsync(c->d_st->phase_ns, 0, sizeof(c->h_st->phase_ns), c->stream);
        c->run_ns_dirty = 0;
    }
    const int e = c->h_st->err;
    if (e & E_CAPACITY) return fail(c, GBEES_ERR_CAPACITY, "cell pool capacity (opts.max_cells) exceeded");
    if (e & E_TABLE_FULL) return fail(c, GBEES_ERR_CAPACITY, "hashtable full");
    if (e & E_KEY_RANGE) return fail(c, GBEES_ERR_KEY_RANGE, "a cell coordinate left the packable key range");
    if (e & E_DEGENERATE) return fail(c, GBEES_ERR_DEGENERATE, "degenerate state (mass <= 0 / non-finite, duplicate key, or no time-step bound)");
    return GBEES_OK;
}

// table clear + insert all + adjacency for all + sum; finish mode as in k_finish
int rebuild_all(gbees_ctx* c, int finish_mode) {
    phase(c, GBEES_PH_REBUILD, 3, [&] {
        k_set_slots<<<1, 1, 0, c->stream>>>(c->p, c->d_st);
        k_clear_table<<<c->grid, TPB, 0, c->stream>>>(c->pool, c->d_st);
        k_rebuild<<<c->grid, TPB, 0, c->stream>>>(c->p, c->pool, c->d_st);
    });
    int rc = GBEES_OK;
    phase(c, GBEES_PH_RELINK, 1, [&] {
        rc = dispatch(c, [&](auto N_, auto D_) {
            k_link<decltype(N_)::value, decltype(D_)::value, true><<<c->grid, TPB, 0, c->stream>>>(c->p, c->pool, c->d_st);
            return GBEES_OK;
        });
    });
    if (rc) return fail(c, rc, "unsupported (n, dynamics) pair");
    phase(c, GBEES_PH_SUM, 2, [&] {
        k_sum<<<c->grid, TPB, 0, c->stream>>>(c->p, c->pool, c->d_st);
        k_finish<<<1, TPB, 0, c->stream>>>(c->p, c->pool, c->d_st, c->grid, finish_mode);
    });
    CU(cudaGetLastError());
    return GBEES_OK;
}

}  // namespace

// ================================================================================================
extern "C" {

int gbees_default_opts(gbees_opts* o) {
    if (!o) return GBEES_ERR_ARG;
    std::memset(o, 0, sizeof(*o));
    o->max_cells = 1 << 20;
    o->load_factor = 0.5;
    o->cfl = 0.9;
    o->hi_res = 1;
    return GBEES_OK;
}

int gbees_destroy(gbees_ctx* c) {
    if (!c) return GBEES_OK;
    cudaSetDevice(c->device);
    cudaStreamSynchronize(c->stream);
    drain_events(c);
    for (cudaEvent_t e : c->ev_free) cudaEventDestroy(e);
    for (int i = 0; i < c->nallocs; ++i) cudaFree(c->allocs[i]);
    if (c->h_st) cudaFreeHost(c->h_st);
    delete c;
    return GBEES_OK;
}

int gbees_create(gbees_ctx** out, int n, const double* dx, double threshold, int dynamics_id,
                 const double* params, int n_params, const gbees_opts* opts_in) {
    if (!out || !dx || n < 1 || n > MAXN) return GBEES_ERR_ARG;
    gbees_opts o;
    gbees_default_opts(&o);
    if (opts_in) o = *opts_in;
    if (o.max_cells <= 0) o.max_cells = 1 << 20;
    if (!(o.load_factor > 0.0 && o.load_factor < 1.0)) o.load_factor = 0.5;
    if (!(o.cfl > 0.0)) o.cfl = 0.9;
    if (o.max_cells >= (int64_t)NBR_TAG) return GBEES_ERR_ARG;
    const int need = dynamics_id == 0 || dynamics_id == 1 ? 3 : dynamics_id == 2 ? 1 : dynamics_id == 3 ? n * n : n;
    if (dynamics_id < 0 || dynamics_id > 4 || n_params < need || (need && !params)) return GBEES_ERR_ARG;
    if ((dynamics_id <= 1 && n != 3) || (dynamics_id == 2 && n < 4)) return GBEES_ERR_ARG;
    for (int j = 0; j < n; ++j) if (!(dx[j] > 0.0)) return GBEES_ERR_ARG;

    gbees_ctx* c = new gbees_ctx();
    c->device = o.device;
    c->stream = (cudaStream_t)o.stream;
    c->no_grow = o.no_grow;
    c->run_mode = o.run_mode;
    Params& p = c->p;
    p.n = n; p.dyn = dynamics_id;
    p.bits = 63 / n > 31 ? 31 : 63 / n;
    p.bias = 1ll << (p.bits - 1);
    p.hi_res = o.hi_res; p.limiter = o.limiter; p.normalise = !o.no_normalise;
    for (int j = 0; j < n; ++j) p.h[j] = dx[j];
    for (int k = 0; k < need; ++k) p.par[k] = params[k];
    p.thresh = threshold; p.cfl = o.cfl;
    p.cap = (uint32_t)o.max_cells;
    p.slots = (uint64_t)std::ceil((double)o.max_cells / o.load_factor);
    p.load_factor = o.load_factor;

    auto bail = [&](int code, const std::string& m) { fprintf(stderr, "gbees_create: %s\n", m.c_str()); gbees_destroy(c); return code; };
    cudaError_t e = cudaSetDevice(c->device);
    if (e != cudaSuccess) return bail(GBEES_ERR_CUDA, cudaGetErrorString(e));
    cudaDeviceProp prop;
    if ((e = cudaGetDeviceProperties(&prop, c->device)) != cudaSuccess) return bail(GBEES_ERR_CUDA, cudaGetErrorString(e));
    c->sms = prop.multiProcessorCount;
    c->grid = (unsigned)c->sms * 8u;
    c->grid_passA = (unsigned)c->sms * 10u;
    c->ntiles_max = (p.cap + SCAN_TILE - 1) / SCAN_TILE;
    const size_t cap = p.cap;
    auto alloc = [&](void** ptr, size_t bytes) {
        cudaError_t e2 = cudaMalloc(ptr, bytes);
        if (e2 == cudaSuccess) c->allocs[c->nallocs++] = *ptr;
        return e2;
    };
    Pool& pl = c->pool;
    if (alloc((void**)&pl.key, cap * 8) || alloc((void**)&pl.Q, cap * 8) || alloc((void**)&pl.acc, cap * 8) ||
        alloc((void**)&pl.mask, cap * 2) || alloc((void**)&pl.nbr, cap * 4 * 2 * n) ||
        alloc((void**)&pl.phi, cap * 8 * 2 * n) || alloc((void**)&pl.table, p.slots * sizeof(ulonglong2)) ||
        alloc((void**)&pl.nbr2, cap * 4 * 2 * n) || alloc((void**)&pl.newidx, cap * 4) ||
        alloc((void**)&pl.key2, cap * 8) || alloc((void**)&pl.Q2, cap * 8) || alloc((void**)&pl.keep, cap) ||
        alloc((void**)&pl.tile_state, (size_t)(c->ntiles_max + 1) * 8) || alloc((void**)&pl.partial, (size_t)c->grid * 8) ||
        alloc((void**)&c->d_st, sizeof(DevState)))
        return bail(GBEES_ERR_CUDA, std::string("cudaMalloc: ") + cudaGetErrorString(cudaGetLastError()));
    if (cudaMallocHost((void**)&c->h_st, sizeof(DevState)) != cudaSuccess) return bail(GBEES_ERR_CUDA, "cudaMallocHost");
    std::memset(c->h_st, 0, sizeof(DevState));
    c->h_st->scale = 1.0;
    cudaMemcpyAsync(c->d_st, c->h_st, sizeof(DevState), cudaMemcpyHostToDevice, c->stream);
    if ((e = cudaStreamSynchronize(c->stream)) != cudaSuccess) return bail(GBEES_ERR_CUDA, cudaGetErrorString(e));
    *out = c;
    return GBEES_OK;
}

const char* gbees_last_error(gbees_ctx* c) { return c ? c->err.c_str() : "null context"; }

int gbees_clear_error(gbees_ctx* c) {
    if (!c) return GBEES_ERR_ARG;
    c->sticky = 0; c->err.clear();
    c->h_st->err = 0;
    cudaSetDevice(c->device);
    cudaMemsetAsync(&c->d_st->err, 0, sizeof(int), c->stream);
    return GBEES_OK;
}

static int reset_state(gbees_ctx* c, uint32_t N) {
    DevState z;
    std::memset(&z, 0, sizeof(z));
    z.N = N; z.scale = 1.0;
    *c->h_st = z;
    CU(cudaMemcpyAsync(c->d_st, c->h_st, sizeof(DevState), cudaMemcpyHostToDevice, c->stream));
    c->n_inserted = c->n_pruned = 0;
    return GBEES_OK;
}

int gbees_init_gaussian(gbees_ctx* c, const double* mean, const double* cov) {
    if (!c || !mean || !cov) return GBEES_ERR_ARG;
    if (c->sticky) return c->sticky;
    CU(cudaSetDevice(c->device));
    const int n = c->p.n;
    GaussArgs g;
    std::memset(&g, 0, sizeof(g));
    double det;
    if (!spd_inverse(n, cov, g.inv, &det)) return GBEES_ERR_NOT_SPD;  // not sticky: caller may retry
    double vol = 1.0;
    for (int j = 0; j < n; ++j) { c->p.mu[j] = mean[j]; vol *= c->p.h[j]; }
    g.norm = vol / std::sqrt(std::pow(2.0 * M_PI, n) * det);
    if (!(g.norm >= c->p.thresh)) return fail(c, GBEES_ERR_DEGENERATE, "threshold above the peak cell mass: empty grid");
    const double r2 = 2.0 * std::log(g.norm / c->p.thresh);
    long double total = 1;
    for (int j = 0; j < n; ++j) {
        g.R[j] = (int64_t)std::floor(std::sqrt(r2 * cov[j * n + j]) / c->p.h[j]) + 1;
        total *= (long double)(2 * g.R[j] + 1);
    }
    if (total > 9.0e18L) return fail(c, GBEES_ERR_CAPACITY, "initial bounding box too large");
    g.total = (unsigned long long)total;
    int rc = reset_state(c, 0);
    if (rc) return rc;
    unsigned long long blocks = (g.total + TPB - 1) / TPB;
    const unsigned grid = (unsigned)(blocks < (unsigned long long)c->sms * 64 ? (blocks ? blocks : 1) : (unsigned long long)c->sms * 64);
    dispatch_n(c, [&](auto N_) {
        k_init_gaussian<decltype(N_)::value><<<grid, TPB, 0, c->stream>>>(c->p, c->pool, c->d_st, g);
        return GBEES_OK;
    });
    if ((rc = sync_state(c))) return rc;   // capacity / range errors before touching the table
    if ((rc = rebuild_all(c, 1))) return rc;
    return sync_state(c);
}

int gbees_import(gbees_ctx* c, const double* origin, const int32_t* keys, const double* pvals, int64_t count) {
    if (!c || !origin || !keys || !pvals || count < 0) return GBEES_ERR_ARG;
    if (c->sticky) return c->sticky;
    if (count > (int64_t)c->p.cap) return fail(c, GBEES_ERR_CAPACITY, "import larger than opts.max_cells");
    CU(cudaSetDevice(c->device));
    const int n = c->p.n;
    for (int j = 0; j < n; ++j) c->p.mu[j] = origin[j];
    // stage through phi / acc (device-to-device or host-to-device, cudaMemcpyDefault picks)
    int32_t* dk = reinterpret_cast<int32_t*>(c->pool.phi);
    double* dp = c->pool.acc;
    CU(cudaMemcpyAsync(dk, keys, (size_t)count * n * 4, cudaMemcpyDefault, c->stream));
    CU(cudaMemcpyAsync(dp, pvals, (size_t)count * 8, cudaMemcpyDefault, c->stream));
    int rc = reset_state(c, (uint32_t)count);
    if (rc) return rc;
    dispatch_n(c, [&](auto N_) {
        k_import<decltype(N_)::value><<<c->grid, TPB, 0, c->stream>>>(c->p, c->pool, c->d_st, dk, dp, (uint32_t)count);
        return GBEES_OK;
    });
    if ((rc = rebuild_all(c, 2))) return rc;
    return sync_state(c);
}

int gbees_step(gbees_ctx* c, double* dt) {
    if (!c || !dt) return GBEES_ERR_ARG;
    if (c->sticky) return c->sticky;
    CU(cudaSetDevice(c->device));
    if (c->h_st->N == 0) return fail(c, GBEES_ERR_DEGENERATE, "empty grid");
    const uint32_t n_before = c->h_st->N;
    int rc = dispatch(c, [&](auto N_, auto D_) {
        constexpr int NN = decltype(N_)::value, DD = decltype(D_)::value;
        phase(c, GBEES_PH_GROW, c->no_grow ? 1 : 2, [&] {
            k_begin<<<1, 1, 0, c->stream>>>(c->d_st, *dt);
            if (!c->no_grow) k_grow<NN, DD><<<c->grid, TPB, 0, c->stream>>>(c->p, c->pool, c->d_st);
        });
        if (!c->no_grow)
            phase(c, GBEES_PH_LINK, 1, [&] { k_link<NN, DD, false><<<c->grid, TPB, 0, c->stream>>>(c->p, c->pool, c->d_st); });
        phase(c, GBEES_PH_PASSA, 1, [&] { k_passA<NN, DD><<<c->grid_passA, PassACfg<NN>::BLK, 0, c->stream>>>(c->p, c->pool, c->d_st); });
        phase(c, GBEES_PH_PASSB, 2, [&] {
            k_passB<NN><<<c->grid, TPB, 0, c->stream>>>(c->p, c->pool, c->d_st);
            k_finish<<<1, TPB, 0, c->stream>>>(c->p, c->pool, c->d_st, c->grid, 0);
        });
        return GBEES_OK;
    });
    if (rc) return fail(c, rc, "unsupported (n, dynamics) pair");
    CU(cudaGetLastError());
    if ((rc = sync_state(c))) return rc;
    c->n_inserted = (int64_t)c->h_st->N - (int64_t)n_before;
    *dt = c->h_st->dt;
    if ((double)c->h_st->N > c->p.load_factor * (double)c->h_st->slots && c->h_st->slots < c->p.slots) {
        // the grid outgrew the active table: rehash into a larger one (adjacency is unaffected)
        phase(c, GBEES_PH_REBUILD, 3, [&] {
            k_set_slots<<<1, 1, 0, c->stream>>>(c->p, c->d_st);
            k_clear_table<<<c->grid, TPB, 0, c->stream>>>(c->pool, c->d_st);
            k_rebuild<<<c->grid, TPB, 0, c->stream>>>(c->p, c->pool, c->d_st);
        });
        // k_set_slots also reset the running CFL maximum: restore it (autonomous f: unchanged by a rehash)
        CU(cudaMemcpyAsync(&c->d_st->smax_bits, &c->h_st->smax_bits, 8, cudaMemcpyHostToDevice, c->stream));
        if ((rc = sync_state(c))) return rc;
    }
    return GBEES_OK;
}

int gbees_prune(gbees_ctx* c) {
    if (!c) return GBEES_ERR_ARG;
    if (c->sticky) return c->sticky;
    CU(cudaSetDevice(c->device));
    const uint32_t N = c->h_st->N;
    if (N == 0) return fail(c, GBEES_ERR_DEGENERATE, "empty grid");
    int rc = GBEES_OK;
    phase(c, GBEES_PH_MARK, 2, [&] {
        cudaMemsetAsync(c->pool.keep, 0, N, c->stream);
        rc = dispatch(c, [&](auto N_, auto D_) {
            k_mark<decltype(N_)::value, decltype(D_)::value><<<c->grid, TPB, 0, c->stream>>>(c->p, c->pool, c->d_st);
            return GBEES_OK;
        });
    });
    if (rc) return fail(c, rc, "unsupported (n, dynamics) pair");
    phase(c, GBEES_PH_COMPACT, 4, [&] {
        cudaMemsetAsync(c->pool.tile_state, 0, (size_t)((N + SCAN_TILE - 1) / SCAN_TILE + 1) * 8, c->stream);
        cudaMemsetAsync(&c->d_st->tile_counter, 0, sizeof(unsigned), c->stream);
        k_compact<<<c->grid, TPB, 0, c->stream>>>(c->p, c->pool, c->d_st);
        k_after_compact<<<1, 1, 0, c->stream>>>(c->p, c->d_st);
    });
    phase(c, GBEES_PH_RELINK, 1, [&] { k_remap_clear<<<c->grid, TPB, 0, c->stream>>>(c->p, c->pool, c->d_st); });
    std::swap(c->pool.key, c->pool.key2);
    std::swap(c->pool.Q, c->pool.Q2);
    std::swap(c->pool.nbr, c->pool.nbr2);
    phase(c, GBEES_PH_REBUILD, 2, [&] {
        rc = dispatch(c, [&](auto N_, auto D_) {
            k_rebuild_smax_sum<decltype(N_)::value, decltype(D_)::value><<<c->grid, TPB, 0, c->stream>>>(c->p, c->pool, c->d_st);
            return GBEES_OK;
        });
        k_finish<<<1, TPB, 0, c->stream>>>(c->p, c->pool, c->d_st, c->grid, 1);
    });
    CU(cudaGetLastError());
    if ((rc = sync_state(c))) return rc;
    c->n_pruned = (int64_t)N - (int64_t)c->h_st->N;
    if (c->h_st->N == 0) return fail(c, GBEES_ERR_DEGENERATE, "prune removed every cell");
    return GBEES_OK;
}

int gbees_correct(gbees_ctx* c, const double* z, const double* R) {
    if (!c || !z || !R) return GBEES_ERR_ARG;
    if (c->sticky) return c->sticky;
    CU(cudaSetDevice(c->device));
    GaussArgs g;
    std::memset(&g, 0, sizeof(g));
    double det;
    if (!spd_inverse(c->p.n, R, g.inv, &det)) return GBEES_ERR_NOT_SPD;
    for (int j = 0; j < c->p.n; ++j) g.v[j] = z[j];
    phase(c, GBEES_PH_CORRECT, 3, [&] {
        dispatch_n(c, [&](auto N_) {
            k_correct<decltype(N_)::value><<<c->grid, TPB, 0, c->stream>>>(c->p, c->pool, c->d_st, g);
            return GBEES_OK;
        });
        k_sum<<<c->grid, TPB, 0, c->stream>>>(c->p, c->pool, c->d_st);
        k_finish<<<1, TPB, 0, c->stream>>>(c->p, c->pool, c->d_st, c->grid, 1);
    });
    CU(cudaGetLastError());
    return sync_state(c);
}

int gbees_export(gbees_ctx* c, int32_t* keys, double* pv, int64_t cap, int64_t* count) {
    if (!c) return GBEES_ERR_ARG;
    if (c->sticky) return c->sticky;
    const int64_t N = c->h_st->N;
    if (count) *count = N;
    if (!keys && !pv) return GBEES_OK;
    if (cap < N) return GBEES_ERR_BUFFER;
    if (N == 0) return GBEES_OK;
    CU(cudaSetDevice(c->device));
    auto on_device = [](const void* ptr) {
        cudaPointerAttributes a;
        if (cudaPointerGetAttributes(&a, ptr) != cudaSuccess) { cudaGetLastError(); return false; }
        return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
    };
    const int n = c->p.n;
    int32_t* dk = keys ? (on_device(keys) ? keys : reinterpret_cast<int32_t*>(c->pool.phi)) : nullptr;
    double* dp = pv ? (on_device(pv) ? pv : c->pool.acc) : nullptr;
    dispatch_n(c, [&](auto N_) {
        k_export<decltype(N_)::value><<<c->grid, TPB, 0, c->stream>>>(c->p, c->pool, c->d_st, dk, dp);
        return GBEES_OK;
    });
    CU(cudaGetLastError());
    if (keys && dk != keys) CU(cudaMemcpyAsync(keys, dk, (size_t)N * n * 4, cudaMemcpyDeviceToHost, c->stream));
    if (pv && dp != pv) CU(cudaMemcpyAsync(pv, dp, (size_t)N * 8, cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    return GBEES_OK;
}

// host loop over gbees_step / gbees_prune: the reference behaviour of gbees_run (opts.run_mode = 1)
static int run_host_loop(gbees_ctx* c, double t_target, int64_t max_steps, int prune_every, int64_t* steps_done) {
    int64_t k = 0;
    int rc = GBEES_OK;
    while (k < max_steps && c->h_st->t < t_target) {
        double dt = t_target < 1e299 ? t_target - c->h_st->t : 0.0;
        if ((rc = gbees_step(c, &dt))) break;
        ++k;
        if (prune_every > 0 && k % prune_every == 0 && (rc = gbees_prune(c))) break;
    }
    if (steps_done) *steps_done = k;
    return rc;
}

int gbees_run(gbees_ctx* c, double t_target, int64_t max_steps, int prune_every, int64_t* steps_done) {
    if (!c) return GBEES_ERR_ARG;
    if (c->sticky) return c->sticky;
    if (steps_done) *steps_done = 0;
    if (c->run_mode == 1) return run_host_loop(c, t_target, max_steps, prune_every, steps_done);
    CU(cudaSetDevice(c->device));
    if (c->h_st->N == 0) return fail(c, GBEES_ERR_DEGENERATE, "empty grid");
    if (max_steps <= 0 || !(c->h_st->t < t_target)) return GBEES_OK;
    const unsigned long long steps0 = c->h_st->steps;
    const unsigned parity0 = c->h_st->parity;
    RunArgs a{t_target, (long long)max_steps, prune_every, c->no_grow};
    int rc = GBEES_OK;
    phase(c, GBEES_PH_RUN, 1, [&] {
        rc = dispatch(c, [&](auto N_, auto D_) {
            auto kern = k_run<decltype(N_)::value, decltype(D_)::value>;
            if (c->run_blocks_per_sm == 0) {
                int nb = 0;
                if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, kern, TPB, 0) != cudaSuccess || nb < 1) return GBEES_ERR_CUDA;
                c->run_blocks_per_sm = nb;
            }
            void* args[] = {(void*)&c->p, (void*)&c->pool, (void*)&c->d_st, (void*)&a};
            cudaError_t e = cudaLaunchCooperativeKernel((void*)kern, dim3((unsigned)(c->sms * c->run_blocks_per_sm)), dim3(TPB),
                                                        args, 0, c->stream);
            return e == cudaSuccess ? GBEES_OK : GBEES_ERR_CUDA;
        });
    });
    if (rc == GBEES_ERR_CUDA) return fail(c, rc, std::string("cooperative launch: ") + cudaGetErrorString(cudaGetLastError()));
    if (rc) return fail(c, rc, "unsupported (n, dynamics) pair");
    rc = sync_state(c);
    if ((c->h_st->parity ^ parity0) & 1u) {   // odd number of prunes inside the loop: buffers swapped
        std::swap(c->pool.key, c->pool.key2);
        std::swap(c->pool.Q, c->pool.Q2);
        std::swap(c->pool.nbr, c->pool.nbr2);
    }
    if (steps_done) *steps_done = (int64_t)(c->h_st->steps - steps0);
    if (rc) return rc;
    if (c->h_st->N == 0) return fail(c, GBEES_ERR_DEGENERATE, "prune removed every cell");
    return GBEES_OK;
}

int gbees_count(gbees_ctx* c, int64_t* count) {
    if (!c || !count) return GBEES_ERR_ARG;
    *count = c->h_st->N;
    return GBEES_OK;
}
int gbees_time(gbees_ctx* c, double* t) {
    if (!c || !t) return GBEES_ERR_ARG;
    *t = c->h_st->t;
    return GBEES_OK;
}
int gbees_stats(gbees_ctx* c, gbees_stats_t* s) {
    if (!c || !s) return GBEES_ERR_ARG;
    s->n_cells = c->h_st->N;
    s->n_inserted = c->n_inserted;
    s->n_pruned = c->n_pruned;
    s->steps = (int64_t)c->h_st->steps;
    s->t = c->h_st->t;
    s->dt = c->h_st->dt;
    s->mass = c->h_st->mass;
    s->cell_updates = (int64_t)c->h_st->cell_updates;
    s->table_slots = (int64_t)c->h_st->slots;
    s->launches = c->launches;
    s->cells_inserted = (int64_t)c->h_st->inserted_total;
    s->cells_prune_scanned = (int64_t)c->h_st->prune_scanned;
    s->prunes = (int64_t)c->h_st->prunes;
    return GBEES_OK;
}

int gbees_run_breakdown(gbees_ctx* c, double* phase_ms) {
    if (!c || !phase_ms) return GBEES_ERR_ARG;
    for (int k = 0; k < GBEES_PHASES; ++k) { phase_ms[k] = c->run_phase_ms[k]; c->run_phase_ms[k] = 0.0; }
    return GBEES_OK;
}

int gbees_profile(gbees_ctx* c, int enable, double* phase_ms, int64_t* phase_launches) {
    if (!c) return GBEES_ERR_ARG;
    cudaSetDevice(c->device);
    cudaStreamSynchronize(c->stream);
    drain_events(c);
    for (int k = 0; k < GBEES_PHASES; ++k) {
        if (phase_ms) phase_ms[k] = c->phase_ms[k];
        if (phase_launches) phase_launches[k] = c->phase_launches[k];
        c->phase_ms[k] = 0.0;
        c->phase_launches[k] = 0;
    }
    c->profile = enable;
    return GBEES_OK;
}

}  // extern "C"
