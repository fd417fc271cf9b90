// Host side of the C ABI in include/gbees.h: context, launches, error handling.
// All arithmetic of the method runs in the kernels of gbees_brick.cuh; the host only computes
// the launch-invariant inputs of init_gaussian / correct (an n x n Cholesky inverse, n <= 6).
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <utility>
#include <vector>

#include "../../include/gbees.h"
#include <cooperative_groups.h>

#include "gbees_brick.cuh"

using namespace gbees;

// ------------------------------------------------------------------------------------------------
// __global__ wrappers (one per phase; Params / Store by value in the constant bank)
// ------------------------------------------------------------------------------------------------
#define GP const __grid_constant__ Params p, const __grid_constant__ Store st_in, DevState* ds
#define ST const Store st = resolve(st_in, ds)
// guard: 0 = always run, 1 = part of a step (runs if ds->go), 2 = part of a prune (runs if ds->prune_ok)
// Programmatic dependent launch: the kernels of a step / prune are enqueued with
// cudaLaunchAttributeProgrammaticStreamSerialization, so the blocks of the next kernel may be scheduled
// while the previous one drains. Every kernel first lets ITS dependents go, then waits until the kernel
// before it has completed and flushed its memory -- before it reads anything, the go flag included.
#define PDL_SYNC() do { asm volatile("griddepcontrol.launch_dependents;"); asm volatile("griddepcontrol.wait;" ::: "memory"); } while (0)
#define GUARD(g) PDL_SYNC(); if (((g) == 1 && !ds->go) || ((g) == 2 && !ds->prune_ok)) return

// start of gbees_step: one step with the caller's cap
__global__ void k_begin_step(DevState* ds, double dt_cap) {
    ds->t_target = 1e300;
    ds->step_limit = ds->steps + 1ull;
    begin_step(ds);
    ds->dt_cap = dt_cap;
}
// start of gbees_run: the device decides step by step whether to go on
__global__ void k_begin_run(DevState* ds, double t_target, unsigned long long step_limit) {
    ds->t_target = t_target;
    ds->step_limit = step_limit;
    ds->prune_ok = 0;
    begin_step(ds);
}
__global__ void k_set_prune_ok(DevState* ds) { ds->prune_ok = 1; }
__global__ void __launch_bounds__(TPB) k_detect(GP) { GUARD(1); ST; phase_detect(p, st, ds); }
template <int NDIM, int DYN, bool SKIP>
__global__ void __launch_bounds__(TPB) k_grow(GP) { GUARD(1); ST; phase_targets<NDIM, DYN, true, SKIP>(p, st, ds); }
template <int NDIM, int DYN>
__global__ void __launch_bounds__(TPB) k_mark(GP) { GUARD(2); ST; phase_targets<NDIM, DYN, false>(p, st, ds); }
template <int NDIM, bool ALL>
__global__ void __launch_bounds__(TPB) k_link(GP, int guard) { GUARD(guard); ST; phase_link<NDIM, ALL>(p, st, ds); }
// pass 1 runs FLUX1_WPB warps per block, 2 blocks per SM (register-capped: 65536 / (2 x 32 x FLUX1_WPB) per thread)
constexpr int FLUX1_WPB = 8;
template <int NDIM, int DYN, bool FAST>
__global__ void __launch_bounds__(32 * FLUX1_WPB, 2) k_flux1(GP) { GUARD(1); ST; phase_flux1<NDIM, DYN, FAST>(p, st, ds); }
// pass 2 + finish; a step that does not execute also cancels the prune enqueued behind it
template <int NDIM>
__global__ void __launch_bounds__(TPB, 8) k_flux2(GP) {
    PDL_SYNC();
    if (!ds->go) { if (gtid() == 0) ds->prune_ok = 0; return; }
    ST;
    phase_flux2_finish<NDIM>(p, st, ds);
}
template <int NDIM, int DYN>
__global__ void __launch_bounds__(TPB) k_smax(GP, int guard) { GUARD(guard); ST; phase_smax<NDIM, DYN>(p, st, ds); }
__global__ void __launch_bounds__(TPB) k_sum(GP, int count, int guard) { GUARD(guard); ST; phase_sum(p, st, ds, count != 0); }
// mode: 1 = renormalise (init / correct / prune), 2 = sum only (import)
__global__ void __launch_bounds__(TPB) k_finish(GP, unsigned nparts, int mode, int guard) {
    GUARD(guard);
    ST;
    Params q = p;
    if (mode == 2) q.normalise = 0;
    finish_sum(q, st, ds, nparts, false);
    if (guard == 2 && threadIdx.x == 0) begin_step(ds);   // the prune changed N / NB: refresh the next step's setup
}
__global__ void __launch_bounds__(TPB) k_prune_scan(GP) { GUARD(2); ST; phase_prune_scan(p, st, ds); }
__global__ void __launch_bounds__(TPB) k_prune_move(GP) { GUARD(2); ST; phase_prune_move(p, st, ds); }
// after the move: unused rows back to zero, and the marks / scan descriptors back to zero for the
// next prune (invariant: keep[] and tile_state[] are all-zero outside a prune)
__device__ __forceinline__ void phase_zero_after_move(const Params& p, const Store& st, DevState* ds) {
    phase_zero_tail(p, st, ds);
    const uint32_t NB = min(ds->NB, p.capB);
    for (uint32_t i = gtid(); i < NB; i += gthreads()) st.keep[i] = 0ull;
    const uint32_t ntiles = (NB + SCAN_TILE - 1) / SCAN_TILE + 1;
    for (uint32_t i = gtid(); i < ntiles; i += gthreads()) st.tile_state[i] = 0ull;
}
__global__ void __launch_bounds__(TPB) k_zero_tail(GP) { GUARD(2); ST; phase_zero_after_move(p, st, ds); }
// prune tail, one launch: re-insert the brick keys, CFL maximum, mass sum + cell count
template <int NDIM, int DYN>
__global__ void __launch_bounds__(TPB) k_prune_tail(GP) {
    GUARD(2);
    ST;
    phase_rebuild(p, st, ds);
    phase_smax<NDIM, DYN>(p, st, ds);
    phase_sum(p, st, ds, true);
}
// adjacency of all bricks; the last block to finish renormalises and sets up the next step
template <int NDIM>
__global__ void __launch_bounds__(TPB) k_link_finish(GP, unsigned nparts) {
    GUARD(2);
    ST;
    __shared__ bool s_last;
    phase_link<NDIM, true>(p, st, ds);
    if (threadIdx.x == 0) {
        __threadfence();
        s_last = atomicAdd(&ds->ticket, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (s_last) {
        __threadfence();
        finish_sum(p, st, ds, nparts, false);
        if (threadIdx.x == 0) { ds->ticket = 0; begin_step(ds); }
    }
}
// after the move: survivors live in Qn and in the second metadata buffers -> flip both parities
__device__ __forceinline__ void after_compact(const Params& p, DevState* ds) {
    ds->prune_scanned += ds->N;
    ds->prunes += 1;
    ds->NB = ds->NB_after_prune;
    ds->NB_before_grow = ds->NB;
    ds->slots = table_slots_for(p, ds->NB);
    ds->smax_bits = 0ull;
    ds->N = 0ull;                      // recounted by k_sum
    ds->tile_counter = 0u;
    ds->parity ^= 3u;
}
__global__ void k_after_compact(const __grid_constant__ Params p, DevState* ds) { GUARD(2); after_compact(p, ds); }

// ---- a9: persistent step loop for SMALL grids -----------------------------------
// While the grid has at most a few hundred bricks a step is pure launch / barrier latency (the paper
// found the same: all its GPUs tie on Lorenz '63). Then the whole loop -- grow, link, pass 1, pass 2,
// prune -- runs in ONE launch of a single thread-block cluster; the hardware cluster barrier
// (barrier.cluster, which also invalidates L1) separates the phases instead of kernel boundaries.
// Same phases, same order, same arithmetic as the stream of launches; leaves the loop when the run
// is over or the grid has outgrown the cluster (the host then goes on with the launches).
// GRID = true is the same loop for grids of any size as ONE cooperative launch that fills the GPU, with
// grid-wide barriers between the phases: the paper's own execution model. It is kept as
// opts.run_mode = 3 for measurement; the stream of launches is faster.
template <int NDIM, int DYN, bool FAST, bool GRID>
__global__ void __launch_bounds__(TPB) k_run_small(GP, int prune_every, int no_grow, unsigned long long k_start, uint32_t nb_limit) {
    namespace cg = cooperative_groups;
    struct Barrier {
        __device__ void sync() const {
            if constexpr (GRID) cg::this_grid().sync();
            else cg::this_cluster().sync();
        }
    } cl;
    __shared__ bool s_last;
    unsigned long long k = k_start;
    for (;;) {
        cl.sync();
        if (GRID && (double)ds->NB_before_grow > p.load_factor * (double)ds->slots && ds->slots < p.slots) break;   // the host rehashes
        // uniform: go and NB_before_grow (= NB at the top of the loop) are written by begin_step only, i.e.
        // before this barrier; NB itself is bumped by the grow below and must not be tested here
        if (!ds->go || ds->NB_before_grow > nb_limit) break;
        Store st = resolve(st_in, ds);
        if (!no_grow) {
            phase_detect(p, st, ds);
            cl.sync();
            phase_targets<NDIM, DYN, true, false>(p, st, ds);
            cl.sync();
            phase_link<NDIM, false>(p, st, ds);
            cl.sync();
        }
        phase_flux1<NDIM, DYN, FAST>(p, st, ds);
        cl.sync();
        phase_flux2_finish<NDIM>(p, st, ds);
        ++k;
        if (prune_every <= 0 || k % (unsigned long long)prune_every != 0) continue;
        cl.sync();
        st = resolve(st_in, ds);                         // the step flipped the Q / Qn parity
        phase_targets<NDIM, DYN, false>(p, st, ds);
        cl.sync();
        phase_prune_scan(p, st, ds);
        cl.sync();
        // (the counts are final after the scan: snapshot them before the barrier that ends the move)
        const uint32_t nb_old = min(ds->NB, p.capB), nb_new = ds->NB_after_prune;
        const unsigned long long new_slots = table_slots_for(p, nb_new);
        phase_prune_move(p, st, ds);
        cl.sync();
        {   // one phase instead of three: zero the vacated rows / marks, update the state, clear the
            // resized table. Everybody works from the snapshot, only thread 0 writes the state.
            for (uint64_t i = (uint64_t)nb_new * 64 + gtid(); i < (uint64_t)nb_old * 64; i += gthreads()) { st.Q[i] = 0.0; st.Qn[i] = 0.0; }
            for (uint32_t i = gtid(); i < nb_old; i += gthreads()) st.keep[i] = 0ull;
            const uint32_t ntiles = (nb_old + SCAN_TILE - 1) / SCAN_TILE + 1;
            for (uint32_t i = gtid(); i < ntiles; i += gthreads()) st.tile_state[i] = 0ull;
            const ulonglong2 e = make_ulonglong2(KEY_EMPTY, KEY_EMPTY);
            for (uint64_t s = gtid(); s < new_slots; s += gthreads()) { st.table[s] = e; st.pend[s] = 0ull; }
            if (gtid() == 0) after_compact(p, ds);
        }
        cl.sync();
        st = resolve(st_in, ds);                         // survivors live in the other buffers now
        phase_rebuild(p, st, ds);
        phase_smax<NDIM, DYN>(p, st, ds);
        phase_sum(p, st, ds, true);
        cl.sync();
        phase_link<NDIM, true>(p, st, ds);
        if (threadIdx.x == 0) {
            __threadfence();
            s_last = atomicAdd(&ds->ticket, 1u) == gridDim.x - 1;
        }
        __syncthreads();
        if (s_last) {
            __threadfence();
            finish_sum(p, st, ds, gridDim.x, false);
            if (threadIdx.x == 0) { ds->ticket = 0; begin_step(ds); }
        }
    }
}
// resize the active table for the current brick count; recount = also reset N and the CFL maximum
__global__ void k_set_slots(const __grid_constant__ Params p, DevState* ds, int recount) {
    ds->slots = table_slots_for(p, min(ds->NB, p.capB));
    if (recount) { ds->smax_bits = 0ull; ds->N = 0ull; }
}
__global__ void __launch_bounds__(TPB) k_clear_table(GP, int guard) { GUARD(guard); ST; phase_clear_table(st, ds); }
__global__ void __launch_bounds__(TPB) k_rebuild(GP, int guard) { GUARD(guard); ST; phase_rebuild(p, st, ds); }
template <int NDIM, bool FILL>
__global__ void __launch_bounds__(TPB) k_init_gaussian(GP, const __grid_constant__ GaussArgs g) {
    ST;
    phase_init_gaussian<NDIM, FILL>(p, st, ds, g);
}
template <int NDIM>
__global__ void __launch_bounds__(TPB) k_correct(GP, const __grid_constant__ GaussArgs g) { ST; phase_correct<NDIM>(p, st, ds, g); }
template <int NDIM>
__global__ void __launch_bounds__(TPB) k_correct_range(GP, const __grid_constant__ GaussArgs g) { ST; phase_correct_range<NDIM>(p, st, ds, g); }
template <int NDIM>
__global__ void __launch_bounds__(TPB) k_correct_linear(GP, const __grid_constant__ GaussArgs g) { ST; phase_correct_linear<NDIM>(p, st, ds, g); }
template <int NDIM>
__global__ void __launch_bounds__(TPB) k_compare(const __grid_constant__ Params p, const __grid_constant__ Store a_in, const DevState* da,
                                                 const __grid_constant__ Store b_in, const DevState* db, double* out) {
    const Store a = resolve(a_in, da), b = resolve(b_in, db);
    phase_compare<NDIM>(p, a, da, b, db, out);
}
// sums the three rows of per-block partials in index order: out3[0..2]
__global__ void __launch_bounds__(TPB) k_compare_finish(const double* part, unsigned nparts, double* out3) {
    for (int q = 0; q < 3; ++q) {
        double v = 0.0;
        for (unsigned k = threadIdx.x; k < nparts; k += blockDim.x) v += part[(size_t)q * nparts + k];
        v = block_sum(v);
        if (threadIdx.x == 0) out3[q] = v;
    }
}
__global__ void __launch_bounds__(TPB) k_marg_clear(unsigned long long* skey, double* sval, unsigned long long S) { phase_marg_clear(skey, sval, S); }
template <int NDIM>
__global__ void __launch_bounds__(TPB) k_marg_accumulate(GP, const __grid_constant__ MargArgs g, unsigned long long* skey, double* sval) {
    ST;
    phase_marg_accumulate<NDIM>(p, st, ds, g, skey, sval);
}
template <int NDIM>
__global__ void __launch_bounds__(TPB) k_resample_accumulate(GP, const __grid_constant__ ResampleArgs g, unsigned long long* skey, double* sval) {
    ST;
    phase_resample_accumulate<NDIM>(p, st, ds, g, skey, sval);
}
__global__ void __launch_bounds__(TPB) k_marg_emit(DevState* ds, const __grid_constant__ MargArgs g, const unsigned long long* skey,
                                                   const double* sval, int32_t* keys, double* out, unsigned cap) {
    phase_marg_emit(ds, g, skey, sval, keys, out, cap);
}
template <int NDIM>
__global__ void __launch_bounds__(TPB) k_export(GP, int32_t* keys, double* out) { ST; phase_export<NDIM>(p, st, ds, keys, out); }
template <int NDIM, bool FILL>
__global__ void __launch_bounds__(TPB) k_import(GP, const int32_t* keys, const double* vals, uint64_t count) {
    ST;
    phase_import<NDIM, FILL>(p, st, ds, keys, vals, count);
}

// ------------------------------------------------------------------------------------------------
// context
// ------------------------------------------------------------------------------------------------
struct gbees_ctx {
    Params p{};
    Store st{};
    DevState* d_st = nullptr;
    DevState* h_st = nullptr;  // pinned mirror
    cudaStream_t stream = nullptr;
    int device = 0;
    int sms = 148;
    unsigned grid = 148 * 8;
    unsigned grid_flux1 = 148 * 2;   // pass 1 (128 registers: 2 resident blocks per SM)
    unsigned ntiles_max = 0;
    size_t stage_bytes = 0;      // size of the phi array (staging area of import / host export)
    int sticky = 0;
    int no_grow = 0;
    int run_mode = 0;            // 0 = device-side step control, 1 = host loop over step/prune
    int small_ok = 1;            // the single-cluster persistent loop can be launched on this device
    int pdl = 1;                 // programmatic dependent launch between the kernels of a step / prune
    cudaGraphExec_t graph_exec = nullptr;   // run_mode 2: the captured chunk
    int64_t graph_chunk = 0;
    int graph_prune = 0;
    int64_t graph_launches = 0;
    int run_blocks_per_sm = 0;
    int64_t n_inserted = 0, n_pruned = 0;
    std::string err;
    void* allocs[32] = {nullptr};
    int nallocs = 0;
    // launch accounting + optional per-phase CUDA-event timing (gbees_profile)
    int64_t launches = 0;
    int profile = 0;
    std::vector<cudaEvent_t> ev_free;
    std::vector<std::pair<int, std::pair<cudaEvent_t, cudaEvent_t>>> ev_open;
    double phase_ms[GBEES_PHASES] = {0};
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

// enqueue one kernel of a step / prune (programmatic dependent launch unless switched off with GBEES_NO_PDL=1)
template <typename... KArgs, typename... Args>
void kl(gbees_ctx* c, void (*kern)(KArgs...), unsigned grid, unsigned block, size_t smem, Args&&... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid); cfg.blockDim = dim3(block); cfg.dynamicSmemBytes = smem; cfg.stream = c->stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = c->pdl;
    cfg.attrs = at; cfg.numAttrs = 1;
    cudaLaunchKernelEx(&cfg, kern, KArgs(std::forward<Args>(args))...);
}

// call f(IC<NDIM>, IC<DYN>) for the context's (n, dynamics) pair; only valid pairs are instantiated
template <typename F>
int dispatch(const gbees_ctx* c, F&& f) {
    const int n = c->p.n, d = c->p.dyn;
#define GB_CASE(N_, D_) if (n == N_ && d == D_) return f(IC<N_>{}, IC<D_>{});
#ifdef GBEES_DEV_PAIRS   // development builds: only the benchmarked pairs (seconds instead of minutes to compile)
    GB_CASE(3, 0) GB_CASE(6, 2) GB_CASE(6, 3)
#else
    GB_CASE(3, 0) GB_CASE(3, 1)
    GB_CASE(4, 2) GB_CASE(5, 2) GB_CASE(6, 2)
    GB_CASE(1, 3) GB_CASE(2, 3) GB_CASE(3, 3) GB_CASE(4, 3) GB_CASE(5, 3) GB_CASE(6, 3)
    GB_CASE(1, 4) GB_CASE(2, 4) GB_CASE(3, 4) GB_CASE(4, 4) GB_CASE(5, 4) GB_CASE(6, 4)
#endif
#undef GB_CASE
    return GBEES_ERR_ARG;
}
template <typename F>
int dispatch_n(const gbees_ctx* c, F&& f) {
    switch (c->p.n) {
#ifndef GBEES_DEV_PAIRS
        case 1: return f(IC<1>{}); case 2: return f(IC<2>{}); case 4: return f(IC<4>{}); case 5: return f(IC<5>{});
#endif
        case 3: return f(IC<3>{}); case 6: return f(IC<6>{});
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
    const int e = c->h_st->err;
    if (e & E_CAPACITY) return fail(c, GBEES_ERR_CAPACITY, "cell pool capacity (opts.max_cells) exceeded");
    if (e & E_TABLE_FULL) return fail(c, GBEES_ERR_CAPACITY, "hashtable full");
    if (e & E_KEY_RANGE) return fail(c, GBEES_ERR_KEY_RANGE, "a cell coordinate left the packable key range");
    if (e & E_DEGENERATE) return fail(c, GBEES_ERR_DEGENERATE, "degenerate state (mass <= 0 / non-finite, duplicate key, or no time-step bound)");
    return GBEES_OK;
}

// after init / import: resize + clear the table, insert all bricks, adjacency for all, CFL maximum,
// mass sum + cell count; finish mode as in k_finish
int rebuild_all(gbees_ctx* c, int finish_mode) {
    phase(c, GBEES_PH_REBUILD, 3, [&] {
        k_set_slots<<<1, 1, 0, c->stream>>>(c->p, c->d_st, 1);
        k_clear_table<<<c->grid, TPB, 0, c->stream>>>(c->p, c->st, c->d_st, 0);
        k_rebuild<<<c->grid, TPB, 0, c->stream>>>(c->p, c->st, c->d_st, 0);
    });
    int rc = GBEES_OK;
    phase(c, GBEES_PH_RELINK, 2, [&] {
        rc = dispatch(c, [&](auto N_, auto D_) {
            k_link<decltype(N_)::value, true><<<c->grid, TPB, 0, c->stream>>>(c->p, c->st, c->d_st, 0);
            k_smax<decltype(N_)::value, decltype(D_)::value><<<c->grid, TPB, 0, c->stream>>>(c->p, c->st, c->d_st, 0);
            return GBEES_OK;
        });
    });
    if (rc) return fail(c, rc, "unsupported (n, dynamics) pair");
    phase(c, GBEES_PH_SUM, 2, [&] {
        k_sum<<<c->grid, TPB, 0, c->stream>>>(c->p, c->st, c->d_st, 1, 0);
        k_finish<<<1, TPB, 0, c->stream>>>(c->p, c->st, c->d_st, c->grid, finish_mode, 0);
    });
    CU(cudaGetLastError());
    return GBEES_OK;
}

// rows [0, NB) of both value buffers back to zero (invariant: unused rows are zero), then a fresh
// state with the whole table allocation in use (the brick count of the new grid is not known yet)
int reset_grid(gbees_ctx* c) {
    const size_t rows = c->h_st->NB < c->p.capB ? c->h_st->NB : c->p.capB;
    if (rows) {
        CU(cudaMemsetAsync(c->st.Q, 0, rows * 64 * 8, c->stream));
        CU(cudaMemsetAsync(c->st.Qn, 0, rows * 64 * 8, c->stream));
    }
    DevState z;
    std::memset(&z, 0, sizeof(z));
    z.scale = 1.0;
    z.slots = c->p.slots;
    *c->h_st = z;
    CU(cudaMemcpyAsync(c->d_st, c->h_st, sizeof(DevState), cudaMemcpyHostToDevice, c->stream));
    k_clear_table<<<c->grid, TPB, 0, c->stream>>>(c->p, c->st, c->d_st, 0);
    c->launches += 1;
    c->n_inserted = c->n_pruned = 0;
    return GBEES_OK;
}

}  // namespace

// ================================================================================================
extern "C" {

// brick and table capacity for (max_cells, load_factor): shared by gbees_create and gbees_arena_bytes
static void plan_capacity(const gbees_opts& o, uint32_t* capB, uint64_t* slots) {
    uint64_t cb = ((uint64_t)o.max_cells + 15) / 16;     // rows of 64 slots; sized for a fill factor >= 1/16
    if (cb < 256) cb = 256;
    *capB = (uint32_t)cb;
    uint64_t s = (uint64_t)std::ceil((double)cb / o.load_factor);
    if (s < (1ull << 16)) s = 1ull << 16;
    *slots = s;
}
constexpr unsigned GRID_MAX = 4096;     // upper bound of c->grid (8 blocks x SMs) used to size the partial-sum array
// device bytes of every fixed-capacity structure, in allocation order (each rounded up to 256 bytes)
static size_t plan_bytes(int n, uint32_t capB, uint64_t slots, size_t* sizes /*[21]*/) {
    const size_t cb = capB, nd = 2 * (size_t)n, ntiles = (capB + SCAN_TILE - 1) / SCAN_TILE;
    const size_t raw[21] = {cb * 512, cb * 512, cb * nd * 32 * 8, cb * 8, cb * 8, cb * 8, cb * 8, cb * 64 * 2, cb * nd * 4,
                            cb * 4, cb * 4, cb * 8, slots * sizeof(ulonglong2), slots * 8, cb * 8, cb * 8, cb * 8, cb * 4,
                            (ntiles + 1) * 8, (size_t)GRID_MAX * 8, sizeof(DevState)};
    size_t tot = 0;
    for (int i = 0; i < 21; ++i) { sizes[i] = (raw[i] + 255) & ~(size_t)255; tot += sizes[i]; }
    return tot;
}

int gbees_arena_bytes(int n, const gbees_opts* opts_in, int64_t* bytes) {
    if (!bytes || n < 1 || n > MAXN) return GBEES_ERR_ARG;
    gbees_opts o;
    gbees_default_opts(&o);
    if (opts_in) o = *opts_in;
    if (o.max_cells <= 0) o.max_cells = 1 << 20;
    if (!(o.load_factor > 0.0 && o.load_factor < 1.0)) o.load_factor = 0.5;
    if (o.max_cells >= (int64_t)1 << 32) return GBEES_ERR_ARG;
    uint32_t capB; uint64_t slots; size_t sizes[21];
    plan_capacity(o, &capB, &slots);
    *bytes = (int64_t)plan_bytes(n, capB, slots, sizes) + 256;    // + alignment slack of the arena's base
    return GBEES_OK;
}

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
    if (c->graph_exec) cudaGraphExecDestroy(c->graph_exec);
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
    if (o.max_cells >= (int64_t)1 << 32) return GBEES_ERR_ARG;   // export / marginal row counters are 32-bit
    const int need = dynamics_id == 0 || dynamics_id == 1 ? 3 : dynamics_id == 2 ? 1 : dynamics_id == 3 ? n * n : n;
    if (dynamics_id < 0 || dynamics_id > 4 || n_params < need || (need && !params)) return GBEES_ERR_ARG;
    if ((dynamics_id <= 1 && n != 3) || (dynamics_id == 2 && n < 4)) return GBEES_ERR_ARG;
    for (int j = 0; j < n; ++j) if (!(dx[j] > 0.0)) return GBEES_ERR_ARG;
    if (!(threshold > 0.0)) return GBEES_ERR_ARG;   // p* > 0: a cell with P = 0 must never be a grow source

    gbees_ctx* c = new gbees_ctx();
    c->device = o.device;
    c->stream = (cudaStream_t)o.stream;
    c->no_grow = o.no_grow;
    c->run_mode = o.run_mode;
    if (const char* e = std::getenv("GBEES_NO_PDL")) c->pdl = !(e[0] == '1');
    Params& p = c->p;
    p.n = n; p.dyn = dynamics_id;
    p.bits = 63 / n > 31 ? 31 : 63 / n;
    p.bias = 1ll << (p.bits - 1);
    p.hi_res = o.hi_res; p.limiter = o.limiter; p.normalise = !o.no_normalise;
    p.h_pow2 = 1;
    for (int j = 0; j < n; ++j) {
        p.h[j] = dx[j];
        p.hinv[j] = 1.0 / dx[j];
        int e;
        if (std::frexp(dx[j], &e) != 0.5) p.h_pow2 = 0;     // mantissa 0.5 <=> power of two
    }
    for (int k = 0; k < need; ++k) p.par[k] = params[k];
    p.thresh = threshold; p.cfl = o.cfl;
    p.max_cells = (uint64_t)o.max_cells;
    plan_capacity(o, &p.capB, &p.slots);
    p.load_factor = o.load_factor;

    auto bail = [&](int code, const std::string& m) { fprintf(stderr, "gbees_create: %s\n", m.c_str()); gbees_destroy(c); return code; };
    cudaError_t e = cudaSetDevice(c->device);
    if (e != cudaSuccess) return bail(GBEES_ERR_CUDA, cudaGetErrorString(e));
    cudaDeviceProp prop;
    if ((e = cudaGetDeviceProperties(&prop, c->device)) != cudaSuccess) return bail(GBEES_ERR_CUDA, cudaGetErrorString(e));
    c->sms = prop.multiProcessorCount;
    c->grid = (unsigned)c->sms * 8u;
    c->grid_flux1 = (unsigned)c->sms * 2u;     // = resident blocks at 128 registers: a persistent grid-stride grid (measured best of 2/4/8/16)
    c->ntiles_max = (p.capB + SCAN_TILE - 1) / SCAN_TILE;
    // dynamic shared memory above 48 KB is an opt-in per function AND per device: set it for this context's device
    if (dispatch(c, [&](auto N_, auto D_) {
            constexpr int NN = decltype(N_)::value, DD = decltype(D_)::value;
            constexpr int smem = (int)(sizeof(Flux1Warp<NN>) * FLUX1_WPB);
            if (cudaFuncSetAttribute(k_flux1<NN, DD, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess ||
                cudaFuncSetAttribute(k_flux1<NN, DD, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess)
                return GBEES_ERR_CUDA;
            return GBEES_OK;
        }) != GBEES_OK)
        return bail(GBEES_ERR_CUDA, "unsupported (n, dynamics) pair or shared-memory opt-in failed");
    const size_t cb = p.capB, nd = 2 * (size_t)n;
    // all fixed-capacity structures: from the caller's arena (opts.arena, carved in 256-byte units) or cudaMalloc
    Store& st = c->st;
    c->stage_bytes = cb * nd * 32 * 8;
    size_t sizes[21];
    const size_t total = plan_bytes(n, p.capB, p.slots, sizes);
    if ((size_t)c->grid > GRID_MAX) return bail(GBEES_ERR_ARG, "more SMs than the partial-sum array is planned for");
    void** const ptrs[21] = {(void**)&st.Q, (void**)&st.Qn, (void**)&st.phi, (void**)&st.bkey, (void**)&st.mask, (void**)&st.grown,
                             (void**)&st.keep, (void**)&st.fetch, (void**)&st.adj, (void**)&st.slot_of, (void**)&st.slist, (void**)&st.smask,
                             (void**)&st.table, (void**)&st.pend, (void**)&st.bkey2, (void**)&st.mask2, (void**)&st.grown2, (void**)&st.newrow,
                             (void**)&st.tile_state, (void**)&st.partial, (void**)&c->d_st};
    if (o.arena) {
        char* base = reinterpret_cast<char*>((reinterpret_cast<uintptr_t>(o.arena) + 255) & ~(uintptr_t)255);
        if (o.arena_bytes < (int64_t)(total + (size_t)(base - reinterpret_cast<char*>(o.arena))))
            return bail(GBEES_ERR_CAPACITY, "opts.arena is smaller than gbees_arena_bytes()");
        for (int i = 0; i < 21; ++i) { *ptrs[i] = base; base += sizes[i]; }
    } else {
        for (int i = 0; i < 21; ++i) {
            if (cudaMalloc(ptrs[i], sizes[i]) != cudaSuccess)
                return bail(GBEES_ERR_CUDA, std::string("cudaMalloc: ") + cudaGetErrorString(cudaGetLastError()));
            c->allocs[c->nallocs++] = *ptrs[i];
        }
    }
    if (cudaMallocHost((void**)&c->h_st, sizeof(DevState)) != cudaSuccess) return bail(GBEES_ERR_CUDA, "cudaMallocHost");
    cudaMemsetAsync(st.Q, 0, cb * 512, c->stream);
    cudaMemsetAsync(st.Qn, 0, cb * 512, c->stream);
    cudaMemsetAsync(st.keep, 0, cb * 8, c->stream);                                    // all-zero outside a prune
    cudaMemsetAsync(st.tile_state, 0, (size_t)(c->ntiles_max + 1) * 8, c->stream);
    std::memset(c->h_st, 0, sizeof(DevState));
    c->h_st->scale = 1.0;
    c->h_st->slots = p.slots;
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
    int rc = reset_grid(c);
    if (rc) return rc;
    unsigned long long blocks = (g.total + TPB - 1) / TPB;
    const unsigned grid = (unsigned)(blocks < (unsigned long long)c->sms * 64 ? (blocks ? blocks : 1) : (unsigned long long)c->sms * 64);
    // two launches: create the bricks, then activate the cells (brick rows are published in between)
    dispatch_n(c, [&](auto N_) {
        k_init_gaussian<decltype(N_)::value, false><<<grid, TPB, 0, c->stream>>>(c->p, c->st, c->d_st, g);
        k_init_gaussian<decltype(N_)::value, true><<<grid, TPB, 0, c->stream>>>(c->p, c->st, c->d_st, g);
        return GBEES_OK;
    });
    c->launches += 2;
    if ((rc = sync_state(c))) return rc;   // capacity / range errors before touching the table
    if ((rc = rebuild_all(c, 1))) return rc;
    return sync_state(c);
}

int gbees_import(gbees_ctx* c, const double* origin, const int32_t* keys, const double* pvals, int64_t count) {
    if (!c || !origin || !keys || !pvals || count < 0) return GBEES_ERR_ARG;
    if (c->sticky) return c->sticky;
    if (count > (int64_t)c->p.max_cells) return fail(c, GBEES_ERR_CAPACITY, "import larger than opts.max_cells");
    CU(cudaSetDevice(c->device));
    const int n = c->p.n;
    for (int j = 0; j < n; ++j) c->p.mu[j] = origin[j];
    // stage through phi (device-to-device or host-to-device, cudaMemcpyDefault picks)
    const size_t kbytes = ((size_t)count * n * 4 + 7) & ~(size_t)7;
    if (kbytes + (size_t)count * 8 > c->stage_bytes) return fail(c, GBEES_ERR_CAPACITY, "import larger than the staging area");
    int32_t* dk = reinterpret_cast<int32_t*>(c->st.phi);
    double* dp = reinterpret_cast<double*>(reinterpret_cast<char*>(c->st.phi) + kbytes);
    if (count) {
        CU(cudaMemcpyAsync(dk, keys, (size_t)count * n * 4, cudaMemcpyDefault, c->stream));
        CU(cudaMemcpyAsync(dp, pvals, (size_t)count * 8, cudaMemcpyDefault, c->stream));
    }
    int rc = reset_grid(c);
    if (rc) return rc;
    dispatch_n(c, [&](auto N_) {
        k_import<decltype(N_)::value, false><<<c->grid, TPB, 0, c->stream>>>(c->p, c->st, c->d_st, dk, dp, (uint64_t)count);
        k_import<decltype(N_)::value, true><<<c->grid, TPB, 0, c->stream>>>(c->p, c->st, c->d_st, dk, dp, (uint64_t)count);
        return GBEES_OK;
    });
    c->launches += 2;
    if ((rc = sync_state(c))) return rc;
    if ((rc = rebuild_all(c, 2))) return rc;
    return sync_state(c);
}

// enqueue the launches of one step (each runs only if the device's go flag is set)
static int enqueue_step(gbees_ctx* c) {
    int rc = dispatch(c, [&](auto N_, auto D_) {
        constexpr int NN = decltype(N_)::value, DD = decltype(D_)::value;
        if (!c->no_grow) {
            phase(c, GBEES_PH_GROW, 2, [&] {
                kl(c, k_detect, c->grid, TPB, 0, c->p, c->st, c->d_st);
                // (large grids list more source bricks than warps fit: throughput variant; small ones: latency variant)
                if (c->h_st->NB > 65536u) kl(c, k_grow<NN, DD, true>, c->grid, TPB, 0, c->p, c->st, c->d_st);
                else kl(c, k_grow<NN, DD, false>, c->grid, TPB, 0, c->p, c->st, c->d_st);
            });
            phase(c, GBEES_PH_LINK, 1, [&] { kl(c, k_link<NN, false>, c->grid, TPB, 0, c->p, c->st, c->d_st, 1); });
        }
        phase(c, GBEES_PH_PASSA, 1, [&] {
            constexpr size_t smem = sizeof(Flux1Warp<NN>) * FLUX1_WPB;   // opt-in above 48 KB: set per device in gbees_create
            if (c->p.hi_res && !c->p.limiter) kl(c, k_flux1<NN, DD, true>, c->grid_flux1, 32 * FLUX1_WPB, smem, c->p, c->st, c->d_st);
            else kl(c, k_flux1<NN, DD, false>, c->grid_flux1, 32 * FLUX1_WPB, smem, c->p, c->st, c->d_st);
        });
        phase(c, GBEES_PH_PASSB, 1, [&] { kl(c, k_flux2<NN>, c->grid, TPB, 0, c->p, c->st, c->d_st); });
        return GBEES_OK;
    });
    if (rc) return fail(c, rc, "unsupported (n, dynamics) pair");
    return GBEES_OK;
}

// enqueue the launches of one prune (each runs only if the device's prune_ok flag is set)
static int enqueue_prune(gbees_ctx* c) {
    int rc = dispatch(c, [&](auto N_, auto D_) {
        constexpr int NN = decltype(N_)::value, DD = decltype(D_)::value;
        phase(c, GBEES_PH_MARK, 1, [&] { kl(c, k_mark<NN, DD>, c->grid, TPB, 0, c->p, c->st, c->d_st); });
        phase(c, GBEES_PH_COMPACT, 4, [&] {
            kl(c, k_prune_scan, c->grid, TPB, 0, c->p, c->st, c->d_st);
            kl(c, k_prune_move, c->grid, TPB, 0, c->p, c->st, c->d_st);
            kl(c, k_zero_tail, c->grid, TPB, 0, c->p, c->st, c->d_st);
            kl(c, k_after_compact, 1, 1, 0, c->p, c->d_st);
        });
        phase(c, GBEES_PH_REBUILD, 2, [&] {
            kl(c, k_clear_table, c->grid, TPB, 0, c->p, c->st, c->d_st, 2);
            kl(c, k_prune_tail<NN, DD>, c->grid, TPB, 0, c->p, c->st, c->d_st);
        });
        phase(c, GBEES_PH_RELINK, 1, [&] { kl(c, k_link_finish<NN>, c->grid, TPB, 0, c->p, c->st, c->d_st, c->grid); });
        return GBEES_OK;
    });
    if (rc) return fail(c, rc, "unsupported (n, dynamics) pair");
    return GBEES_OK;
}

// the grid outgrew the active table: rehash into a larger one (adjacency is unaffected)
static int rehash_if_needed(gbees_ctx* c) {
    if (!((double)c->h_st->NB > c->p.load_factor * (double)c->h_st->slots && c->h_st->slots < c->p.slots)) return GBEES_OK;
    phase(c, GBEES_PH_REBUILD, 3, [&] {
        k_set_slots<<<1, 1, 0, c->stream>>>(c->p, c->d_st, 0);
        k_clear_table<<<c->grid, TPB, 0, c->stream>>>(c->p, c->st, c->d_st, 0);
        k_rebuild<<<c->grid, TPB, 0, c->stream>>>(c->p, c->st, c->d_st, 0);
    });
    return sync_state(c);
}

int gbees_step(gbees_ctx* c, double* dt) {
    if (!c || !dt) return GBEES_ERR_ARG;
    if (c->sticky) return c->sticky;
    CU(cudaSetDevice(c->device));
    if (c->h_st->N == 0) return fail(c, GBEES_ERR_DEGENERATE, "empty grid");
    const unsigned long long n_before = c->h_st->N;
    phase(c, GBEES_PH_GROW, 1, [&] { k_begin_step<<<1, 1, 0, c->stream>>>(c->d_st, *dt); });
    int rc = enqueue_step(c);
    if (rc) return rc;
    CU(cudaGetLastError());
    if ((rc = sync_state(c))) return rc;
    c->n_inserted = (int64_t)c->h_st->N - (int64_t)n_before;
    *dt = c->h_st->dt;
    return rehash_if_needed(c);
}

int gbees_prune(gbees_ctx* c) {
    if (!c) return GBEES_ERR_ARG;
    if (c->sticky) return c->sticky;
    CU(cudaSetDevice(c->device));
    const unsigned long long N = c->h_st->N;
    if (N == 0) return fail(c, GBEES_ERR_DEGENERATE, "empty grid");
    k_set_prune_ok<<<1, 1, 0, c->stream>>>(c->d_st);
    c->launches += 1;
    int rc = enqueue_prune(c);
    if (rc) return rc;
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
            k_correct<decltype(N_)::value><<<c->grid, TPB, 0, c->stream>>>(c->p, c->st, c->d_st, g);
            return GBEES_OK;
        });
        k_sum<<<c->grid, TPB, 0, c->stream>>>(c->p, c->st, c->d_st, 0, 0);
        k_finish<<<1, TPB, 0, c->stream>>>(c->p, c->st, c->d_st, c->grid, 1, 0);
    });
    CU(cudaGetLastError());
    return sync_state(c);
}

int gbees_correct_range(gbees_ctx* c, const double* s, double y, double sigma) {
    if (!c || !s) return GBEES_ERR_ARG;
    if (!(sigma > 0.0)) return GBEES_ERR_NOT_SPD;
    if (c->sticky) return c->sticky;
    CU(cudaSetDevice(c->device));
    GaussArgs g;
    std::memset(&g, 0, sizeof(g));
    for (int j = 0; j < c->p.n; ++j) g.v[j] = s[j];
    g.norm = y;
    g.inv[0] = 1.0 / sigma;
    phase(c, GBEES_PH_CORRECT, 3, [&] {
        dispatch_n(c, [&](auto N_) {
            k_correct_range<decltype(N_)::value><<<c->grid, TPB, 0, c->stream>>>(c->p, c->st, c->d_st, g);
            return GBEES_OK;
        });
        k_sum<<<c->grid, TPB, 0, c->stream>>>(c->p, c->st, c->d_st, 0, 0);
        k_finish<<<1, TPB, 0, c->stream>>>(c->p, c->st, c->d_st, c->grid, 1, 0);
    });
    CU(cudaGetLastError());
    return sync_state(c);
}

int gbees_correct_linear(gbees_ctx* c, const double* H, int m, const double* y, const double* R) {
    if (!c || !H || !y || !R || m < 1 || m > MAXN) return GBEES_ERR_ARG;
    if (c->sticky) return c->sticky;
    CU(cudaSetDevice(c->device));
    GaussArgs g;
    std::memset(&g, 0, sizeof(g));
    double det;
    if (!spd_inverse(m, R, g.inv, &det)) return GBEES_ERR_NOT_SPD;
    g.m = m;
    for (int k = 0; k < m * c->p.n; ++k) g.H[k] = H[k];
    for (int r = 0; r < m; ++r) g.v[r] = y[r];
    phase(c, GBEES_PH_CORRECT, 3, [&] {
        dispatch_n(c, [&](auto N_) {
            k_correct_linear<decltype(N_)::value><<<c->grid, TPB, 0, c->stream>>>(c->p, c->st, c->d_st, g);
            return GBEES_OK;
        });
        k_sum<<<c->grid, TPB, 0, c->stream>>>(c->p, c->st, c->d_st, 0, 0);
        k_finish<<<1, TPB, 0, c->stream>>>(c->p, c->st, c->d_st, c->grid, 1, 0);
    });
    CU(cudaGetLastError());
    return sync_state(c);
}

int gbees_compare(gbees_ctx* c, gbees_ctx* o, double* bc, double* l1) {
    if (!c || !o || !bc || !l1) return GBEES_ERR_ARG;
    if (c->sticky) return c->sticky;
    if (o->sticky) return o->sticky;
    if (c->p.n != o->p.n || c->device != o->device) return GBEES_ERR_ARG;
    for (int j = 0; j < c->p.n; ++j)
        if (c->p.h[j] != o->p.h[j] || c->p.mu[j] != o->p.mu[j]) return GBEES_ERR_ARG;   // same grid only
    CU(cudaSetDevice(c->device));
    CU(cudaStreamSynchronize(o->stream));            // the other context's state is complete
    CU(cudaStreamSynchronize(c->stream));
    double* part = c->st.phi;                          // free between steps: 3 x grid partials + 2 x 3 results
    double* res = part + 3 * (size_t)c->grid;
    dispatch_n(c, [&](auto N_) {
        k_compare<decltype(N_)::value><<<c->grid, TPB, 0, c->stream>>>(c->p, c->st, c->d_st, o->st, o->d_st, part);
        k_compare_finish<<<1, TPB, 0, c->stream>>>(part, c->grid, res);
        k_compare<decltype(N_)::value><<<c->grid, TPB, 0, c->stream>>>(o->p, o->st, o->d_st, c->st, c->d_st, part);   // the scanned side's own capB
        k_compare_finish<<<1, TPB, 0, c->stream>>>(part, c->grid, res + 3);
        return GBEES_OK;
    });
    c->launches += 4;
    CU(cudaGetLastError());
    double h[6];
    CU(cudaMemcpyAsync(h, res, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    *bc = h[0];
    *l1 = h[1] + h[5];     // |Pa - Pb| over this grid's cells + |Pb| over the cells only the other grid has
    return GBEES_OK;
}

int gbees_marginal(gbees_ctx* c, const int* dims, int m, int32_t* keys, double* pv, int64_t cap, int64_t* count) {
    if (!c || !dims || !count || m < 1 || m > c->p.n) return GBEES_ERR_ARG;
    if (c->sticky) return c->sticky;
    MargArgs g;
    std::memset(&g, 0, sizeof(g));
    g.m = m;
    for (int r = 0; r < m; ++r) {
        if (dims[r] < 0 || dims[r] >= c->p.n) return GBEES_ERR_ARG;
        for (int q = 0; q < r; ++q) if (dims[q] == dims[r]) return GBEES_ERR_ARG;
        g.dims[r] = dims[r];
    }
    g.mbits = 63 / m > 32 ? 32 : 63 / m;
    if (g.mbits < c->p.bits) g.mbits = c->p.bits;                 // m <= n, so floor(63/m) >= floor(63/n) anyway
    const unsigned long long N = c->h_st->N;
    if (N == 0) { *count = 0; return GBEES_OK; }
    CU(cudaSetDevice(c->device));
    g.S = 1024;
    while (g.S < 2 * N) g.S <<= 1;                                // at most N marginal cells: load factor <= 0.5
    // scratch in the phi array (free between steps): table keys, table values, then the output staging area
    const size_t need = (size_t)g.S * 16 + (size_t)N * (4 * (size_t)m + 8) + 64;
    if (need > c->stage_bytes) { c->err = "marginal: scratch larger than the staging area"; return GBEES_ERR_CAPACITY; }   // a query: not sticky
    unsigned long long* skey = reinterpret_cast<unsigned long long*>(c->st.phi);
    double* sval = reinterpret_cast<double*>(skey + g.S);
    char* stage = reinterpret_cast<char*>(sval + g.S);
    auto on_device = [](const void* ptr) {
        cudaPointerAttributes a;
        if (cudaPointerGetAttributes(&a, ptr) != cudaSuccess) { cudaGetLastError(); return false; }
        return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
    };
    const bool dev_out = keys && pv && on_device(keys) && on_device(pv);
    const unsigned ucap = keys && pv ? (dev_out ? (unsigned)(cap < (int64_t)N ? cap : (int64_t)N) : (unsigned)N) : 0u;
    const size_t kbytes = ((size_t)N * m * 4 + 7) & ~(size_t)7;
    int32_t* dk = dev_out ? keys : reinterpret_cast<int32_t*>(stage);
    double* dp = dev_out ? pv : reinterpret_cast<double*>(stage + kbytes);
    CU(cudaMemsetAsync(&c->d_st->export_count, 0, sizeof(unsigned), c->stream));
    k_marg_clear<<<c->grid, TPB, 0, c->stream>>>(skey, sval, g.S);
    dispatch_n(c, [&](auto N_) {
        k_marg_accumulate<decltype(N_)::value><<<c->grid, TPB, 0, c->stream>>>(c->p, c->st, c->d_st, g, skey, sval);
        return GBEES_OK;
    });
    k_marg_emit<<<c->grid, TPB, 0, c->stream>>>(c->d_st, g, skey, sval, dk, dp, ucap);
    c->launches += 3;
    CU(cudaGetLastError());
    unsigned got = 0;
    CU(cudaMemcpyAsync(&got, &c->d_st->export_count, sizeof(unsigned), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    *count = got;
    if (!keys || !pv) return GBEES_OK;                            // count only
    if (cap < (int64_t)got) return GBEES_ERR_BUFFER;
    if (!dev_out) {
        CU(cudaMemcpyAsync(keys, dk, (size_t)got * m * 4, cudaMemcpyDeviceToHost, c->stream));
        CU(cudaMemcpyAsync(pv, dp, (size_t)got * 8, cudaMemcpyDeviceToHost, c->stream));
        CU(cudaStreamSynchronize(c->stream));
    }
    return GBEES_OK;
}

int gbees_resample(gbees_ctx* c, const double* origin2, const double* dx2, int32_t* keys, double* pv, int64_t cap, int64_t* count) {
    if (!c || !origin2 || !dx2 || !count) return GBEES_ERR_ARG;
    if (c->sticky) return c->sticky;
    const int n = c->p.n;
    ResampleArgs g;
    std::memset(&g, 0, sizeof(g));
    for (int j = 0; j < n; ++j) {
        if (!(dx2[j] >= c->p.h[j])) return GBEES_ERR_ARG;           // the target grid is at least as coarse in every dimension
        g.o2[j] = origin2[j]; g.h2[j] = dx2[j];
    }
    g.mbits = c->p.bits;
    const unsigned long long N = c->h_st->N;
    if (N == 0) { *count = 0; return GBEES_OK; }
    CU(cudaSetDevice(c->device));
    g.S = 1024;
    while (g.S < 4 * N) g.S <<= 1;                                // a coarser grid has fewer cells than the source: load factor <= 0.25 + halo
    const size_t ocap = (size_t)g.S / 2;                           // output rows staged at most (distinct target cells <= slots in use)
    const size_t need = (size_t)g.S * 16 + ocap * (4 * (size_t)n + 8) + 64;
    if (need > c->stage_bytes) { c->err = "resample: scratch larger than the staging area"; return GBEES_ERR_CAPACITY; }   // a query: not sticky
    unsigned long long* skey = reinterpret_cast<unsigned long long*>(c->st.phi);
    double* sval = reinterpret_cast<double*>(skey + g.S);
    char* stage = reinterpret_cast<char*>(sval + g.S);
    auto on_device = [](const void* ptr) {
        cudaPointerAttributes a;
        if (cudaPointerGetAttributes(&a, ptr) != cudaSuccess) { cudaGetLastError(); return false; }
        return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
    };
    const bool dev_out = keys && pv && on_device(keys) && on_device(pv);
    const unsigned ucap = keys && pv ? (dev_out ? (unsigned)(cap < (int64_t)ocap ? cap : (int64_t)ocap) : (unsigned)ocap) : 0u;
    const size_t kbytes = (ocap * n * 4 + 7) & ~(size_t)7;
    int32_t* dk = dev_out ? keys : reinterpret_cast<int32_t*>(stage);
    double* dp = dev_out ? pv : reinterpret_cast<double*>(stage + kbytes);
    MargArgs e;                                                    // emit: all n target coordinates, in order
    std::memset(&e, 0, sizeof(e));
    e.m = n; e.mbits = g.mbits; e.S = g.S;
    CU(cudaMemsetAsync(&c->d_st->export_count, 0, sizeof(unsigned), c->stream));
    k_marg_clear<<<c->grid, TPB, 0, c->stream>>>(skey, sval, g.S);
    dispatch_n(c, [&](auto N_) {
        k_resample_accumulate<decltype(N_)::value><<<c->grid, TPB, 0, c->stream>>>(c->p, c->st, c->d_st, g, skey, sval);
        return GBEES_OK;
    });
    k_marg_emit<<<c->grid, TPB, 0, c->stream>>>(c->d_st, e, skey, sval, dk, dp, ucap);
    c->launches += 3;
    CU(cudaGetLastError());
    unsigned got = 0;
    CU(cudaMemcpyAsync(&got, &c->d_st->export_count, sizeof(unsigned), cudaMemcpyDeviceToHost, c->stream));
    int rc = sync_state(c);                                        // table-full / finer-grid faults raised on the device
    if (rc) return rc;
    *count = got;
    if (!keys || !pv) return GBEES_OK;                            // count only
    if (cap < (int64_t)got || got > ucap) return GBEES_ERR_BUFFER;
    if (!dev_out) {
        CU(cudaMemcpyAsync(keys, dk, (size_t)got * n * 4, cudaMemcpyDeviceToHost, c->stream));
        CU(cudaMemcpyAsync(pv, dp, (size_t)got * 8, cudaMemcpyDeviceToHost, c->stream));
        CU(cudaStreamSynchronize(c->stream));
    }
    return GBEES_OK;
}

int gbees_export(gbees_ctx* c, int32_t* keys, double* pv, int64_t cap, int64_t* count) {
    if (!c) return GBEES_ERR_ARG;
    if (c->sticky) return c->sticky;
    const int64_t N = (int64_t)c->h_st->N;
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
    // host buffers are served through the phi array (free between steps) as a staging area
    const size_t kbytes = ((size_t)N * n * 4 + 7) & ~(size_t)7;
    if (kbytes + (size_t)N * 8 > c->stage_bytes) return fail(c, GBEES_ERR_CAPACITY, "export larger than the staging area");
    int32_t* dk = keys ? (on_device(keys) ? keys : reinterpret_cast<int32_t*>(c->st.phi)) : nullptr;
    double* dp = pv ? (on_device(pv) ? pv : reinterpret_cast<double*>(reinterpret_cast<char*>(c->st.phi) + kbytes)) : nullptr;
    CU(cudaMemsetAsync(&c->d_st->export_count, 0, sizeof(unsigned), c->stream));
    dispatch_n(c, [&](auto N_) {
        k_export<decltype(N_)::value><<<c->grid, TPB, 0, c->stream>>>(c->p, c->st, c->d_st, dk, dp);
        return GBEES_OK;
    });
    c->launches += 1;
    CU(cudaGetLastError());
    if (keys && dk != keys) CU(cudaMemcpyAsync(keys, dk, (size_t)N * n * 4, cudaMemcpyDeviceToHost, c->stream));
    if (pv && dp != pv) CU(cudaMemcpyAsync(pv, dp, (size_t)N * 8, cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    return GBEES_OK;
}

// small grids: the whole loop in one launch of a single 8-block cluster (k_run_small)
constexpr uint32_t SMALL_NB_ENTER = 256, SMALL_NB_LEAVE = 512;
static int launch_small(gbees_ctx* c, int prune_every, unsigned long long k_start) {
    int rc = dispatch(c, [&](auto N_, auto D_) {
        constexpr int NN = decltype(N_)::value, DD = decltype(D_)::value;
        constexpr size_t smem = sizeof(Flux1Warp<NN>) * WPB;
        const bool fast = c->p.hi_res && !c->p.limiter;
        auto kern = fast ? k_run_small<NN, DD, true, false> : k_run_small<NN, DD, false, false>;
        if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return GBEES_ERR_CUDA;
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(8); cfg.blockDim = dim3(TPB); cfg.dynamicSmemBytes = smem; cfg.stream = c->stream;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = 8; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        cfg.attrs = at; cfg.numAttrs = 1;
        cudaError_t e = cudaSuccess;
        phase(c, GBEES_PH_RUN, 1, [&] {
            e = cudaLaunchKernelEx(&cfg, kern, c->p, c->st, c->d_st, prune_every, c->no_grow, k_start, SMALL_NB_LEAVE);
        });
        return e == cudaSuccess ? GBEES_OK : GBEES_ERR_CUDA;
    });
    if (rc == GBEES_ERR_CUDA) { cudaGetLastError(); c->small_ok = 0; }   // not launchable here: use the launches
    return rc;
}

// opts.run_mode = 3: the whole loop as one cooperative launch over the GPU (measurement; see k_run_small)
static int launch_coop(gbees_ctx* c, int prune_every, unsigned long long k_start) {
    return dispatch(c, [&](auto N_, auto D_) {
        constexpr int NN = decltype(N_)::value, DD = decltype(D_)::value;
        constexpr size_t smem = sizeof(Flux1Warp<NN>) * WPB;
        const bool fast = c->p.hi_res && !c->p.limiter;
        auto kern = fast ? k_run_small<NN, DD, true, true> : k_run_small<NN, DD, false, true>;
        if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return GBEES_ERR_CUDA;
        int per_sm = 0;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, TPB, smem) != cudaSuccess || per_sm < 1) return GBEES_ERR_CUDA;
        Params p = c->p; Store st = c->st; DevState* ds = c->d_st;
        int pe = prune_every, ng = c->no_grow; unsigned long long ks = k_start; uint32_t lim = c->p.capB;
        void* args[] = {&p, &st, &ds, &pe, &ng, &ks, &lim};
        cudaError_t e = cudaSuccess;
        phase(c, GBEES_PH_RUN, 1, [&] {
            e = cudaLaunchCooperativeKernel((const void*)kern, dim3((unsigned)(per_sm * c->sms)), dim3(TPB), args, smem, c->stream);
        });
        return e == cudaSuccess ? GBEES_OK : GBEES_ERR_CUDA;
    });
}

// opts.run_mode = 2: a chunk of steps (+ its prunes) captured once as a CUDA graph and relaunched (measurement).
// The launches are identical from chunk to chunk -- all state is on the device -- as long as the chunk is a
// multiple of the prune cadence.
static int enqueue_step(gbees_ctx* c);
static int enqueue_prune(gbees_ctx* c);
static int launch_graph_chunk(gbees_ctx* c, int64_t chunk, int prune_every) {
    if (!c->graph_exec || c->graph_chunk != chunk || c->graph_prune != prune_every) {
        if (c->graph_exec) { cudaGraphExecDestroy(c->graph_exec); c->graph_exec = nullptr; }
        cudaGraph_t g = nullptr;
        const int64_t l0 = c->launches;
        if (cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) return GBEES_ERR_CUDA;
        int rc = GBEES_OK;
        for (int64_t i = 1; i <= chunk && !rc; ++i) {
            rc = enqueue_step(c);
            if (!rc && prune_every > 0 && i % prune_every == 0) rc = enqueue_prune(c);
        }
        if (cudaStreamEndCapture(c->stream, &g) != cudaSuccess || rc) { if (g) cudaGraphDestroy(g); return rc ? rc : GBEES_ERR_CUDA; }
        const cudaError_t e = cudaGraphInstantiate(&c->graph_exec, g, 0);
        cudaGraphDestroy(g);
        if (e != cudaSuccess) { c->graph_exec = nullptr; return GBEES_ERR_CUDA; }
        c->graph_chunk = chunk; c->graph_prune = prune_every;
        c->graph_launches = c->launches - l0;
        c->launches = l0;
    }
    c->launches += c->graph_launches;
    return cudaGraphLaunch(c->graph_exec, c->stream) == cudaSuccess ? GBEES_OK : GBEES_ERR_CUDA;
}

// host loop over gbees_step / gbees_prune with a host round trip per call (opts.run_mode = 1)
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

// Step loop without host round trips (PAPER.md:170-172 keeps the whole loop on the device; here the
// device decides per step whether the enqueued launches execute, and the host only reads the state
// back once per chunk of steps).
int gbees_run(gbees_ctx* c, double t_target, int64_t max_steps, int prune_every, int64_t* steps_done) {
    if (!c) return GBEES_ERR_ARG;
    if (c->sticky) return c->sticky;
    if (steps_done) *steps_done = 0;
    if (c->run_mode == 1) return run_host_loop(c, t_target, max_steps, prune_every, steps_done);
    CU(cudaSetDevice(c->device));
    if (c->h_st->N == 0) return fail(c, GBEES_ERR_DEGENERATE, "empty grid");
    if (max_steps <= 0 || !(c->h_st->t < t_target)) return GBEES_OK;
    const unsigned long long steps0 = c->h_st->steps;
    const unsigned long long limit = (unsigned long long)max_steps > (~0ull >> 1) - steps0 ? (~0ull >> 1) : steps0 + (unsigned long long)max_steps;
    const unsigned long long n_before = c->h_st->N;
    k_begin_run<<<1, 1, 0, c->stream>>>(c->d_st, t_target, limit);
    c->launches += 1;
    int rc = GBEES_OK;
    int64_t k = 0;     // steps enqueued
    for (;;) {
        if (c->small_ok && !c->profile && c->h_st->NB <= SMALL_NB_ENTER) {
            const int lrc = launch_small(c, prune_every, (unsigned long long)k);
            if (lrc == GBEES_OK) {
                if ((rc = sync_state(c))) break;
                k = (int64_t)(c->h_st->steps - steps0);
                if (!c->h_st->go || k >= max_steps) break;
                if (c->h_st->NB <= SMALL_NB_ENTER) c->small_ok = 0;   // left the loop for another reason: do not spin
                else continue;
            } else if (lrc != GBEES_ERR_CUDA) return fail(c, lrc, "unsupported (n, dynamics) pair");
        }
        if (c->run_mode == 3 && !c->profile) {               // one cooperative launch runs until the end (or a rehash)
            const int lrc = launch_coop(c, prune_every, (unsigned long long)k);
            if (lrc != GBEES_OK) return fail(c, lrc, "cooperative launch failed");
            if ((rc = sync_state(c))) break;
            if ((rc = rehash_if_needed(c))) break;
            k = (int64_t)(c->h_st->steps - steps0);
            if (!c->h_st->go || k >= max_steps) break;
            continue;
        }
        if (c->run_mode == 2 && !c->profile && (prune_every <= 0 || k % prune_every == 0)) {
            const int64_t gchunk = prune_every > 0 ? (int64_t)prune_every * ((16 + prune_every - 1) / prune_every) : 16;
            if (gchunk <= max_steps - k) {
                if ((rc = launch_graph_chunk(c, gchunk, prune_every)))
                    return fail(c, rc, std::string("CUDA graph of a chunk of steps (not capturable on the legacy default stream): ") + cudaGetErrorString(cudaGetLastError()));
                k += gchunk;
                if ((rc = sync_state(c))) break;
                if ((rc = rehash_if_needed(c))) break;
                if (!c->h_st->go || k >= max_steps) break;
                continue;
            }
        }
        int64_t chunk = 16;
        if (c->h_st->dt > 0.0 && t_target < 1e299) {     // do not enqueue far past the expected end
            const double est = (t_target - c->h_st->t) / c->h_st->dt;
            if (est < (double)chunk) chunk = (int64_t)est + 2;
        }
        if (chunk > max_steps - k) chunk = max_steps - k;
        for (int64_t i = 0; i < chunk; ++i) {
            if ((rc = enqueue_step(c))) return rc;
            ++k;
            if (prune_every > 0 && k % prune_every == 0 && (rc = enqueue_prune(c))) return rc;
        }
        CU(cudaGetLastError());
        if ((rc = sync_state(c))) break;
        if ((rc = rehash_if_needed(c))) break;
        if (!c->h_st->go || k >= max_steps) break;
    }
    c->n_inserted = (int64_t)c->h_st->N - (int64_t)n_before;
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
