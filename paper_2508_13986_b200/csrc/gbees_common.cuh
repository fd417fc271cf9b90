// Device-side building blocks of the GBEES prediction step (sm_100a): key packing, hashtable,
// dynamics / face velocities. See DESIGN.md for layout and semantics; citations are PAPER.md lines.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace gbees {

constexpr int MAXN = 6;
constexpr uint64_t KEY_EMPTY = ~0ull;            // all-ones is never a packed key (A18)
constexpr uint32_t NBR_NONE = 0xFFFFFFFFu;       // no neighbour, direct or two-hop

enum ErrBits : int { E_CAPACITY = 1, E_KEY_RANGE = 2, E_DEGENERATE = 4, E_TABLE_FULL = 8 };

// Launch-invariant problem description, passed by value (__grid_constant__) to every kernel.
struct Params {
    int n;
    int dyn;
    int bits;            // bits per coordinate field = min(floor(63/n), 31)
    int hi_res;
    int limiter;
    int normalise;
    int64_t bias;        // 2^(bits-1): cell coordinates live in [-bias, bias-1] (A18)
    double h[MAXN];
    double hinv[MAXN];   // 1 / h_j
    int h_pow2;          // every h_j is a power of two: x / h_j == x * hinv_j bit for bit
    double mu[MAXN];     // grid origin
    double par[MAXN * MAXN];
    double thresh;
    double cfl;
    uint64_t max_cells;  // opts.max_cells: active-cell capacity
    uint32_t capB;       // brick capacity (rows of 64 cell slots)
    uint64_t slots;      // hashtable slots allocated (= ceil(capB / load_factor))
    double load_factor;  // rehash to a larger active table when NB / slots_in_use exceeds this
};

// Mutable scalars living in device memory (one struct, read back after each API call).
struct DevState {
    unsigned long long N;          // active cells
    unsigned long long N_before_grow;
    unsigned long long Ncount;     // active cells counted by pass 1 of the running step
    uint32_t nsrc;                 // bricks with new sources listed by this step's detect (slist / smask)
    uint32_t NB;                   // bricks in use (rows 0..NB-1)
    uint32_t NB_before_grow;       // bricks before this step's grow (link range start)
    int err;
    unsigned int ticket;           // last-block election for the sum reduction
    unsigned long long smax_bits;  // bits of max_c sum_j |u_cj|/h_j  (>= 0, so uint order == fp order)
    double sumQ;                   // sum of stored masses Q
    double scale;                  // P = scale * Q
    double dt;
    double dt_cap;                 // caller's cap for this step (<= 0 / non-finite: none)
    double t;
    double mass;                   // pre-normalisation mass of the last step (in normalised units)
    unsigned long long steps;
    unsigned long long cell_updates;
    unsigned int tile_counter;     // dynamic tile ids for the decoupled-lookback scan
    uint32_t NB_after_prune;
    unsigned long long inserted_total;   // cells created by grow since init
    unsigned long long prune_scanned;    // sum over prunes of the cell count scanned
    unsigned long long prunes;
    unsigned int parity;                 // bit 0 = Q/Qn swapped, bit 1 = metadata double buffers swapped (resolve())
    unsigned int export_count;           // export: next output row
    double t_target;                     // gbees_run: advance until t == t_target ...
    unsigned long long step_limit;       // ... or until steps == step_limit
    int go;                              // the step being enqueued executes (decided on the device by begin_step)
    int prune_ok;                        // the last enqueued step executed: the prune that follows it runs
    unsigned long long slots;            // hashtable slots in use (<= Params::slots), resized at rehash
};

// Brick store. A brick is a dense box of 64 cell slots (2^K_j cells along
// dimension j, sum K_j = 6); row r of the store holds brick r. Inactive slots hold Q = 0.
struct Store {
    double* Q;           // [capB][64] stored mass (P = scale * Q)
    double* Qn;          // [capB][64] next-step buffer (pass 1 partial update, pass 2 final)
    double* phi;         // [capB][2n][32] tau_j * flux through the EXTERNAL faces owned (upwind) by this brick
    uint64_t* bkey;      // [capB] packed brick coordinates
    uint64_t* mask;      // [capB] active-cell bits (bit = local index)
    uint64_t* grown;     // [capB] cells whose Targets(c) have been inserted (autonomous f: grow once)
    uint64_t* keep;      // [capB] prune marks
    uint16_t* fetch;     // [capB][64] per cell: bit d = fetch the flux of external face d from the neighbour brick in pass 2
    uint32_t* adj;       // [capB][2n] neighbour brick rows: d = 2j (-e^j), 2j+1 (+e^j); NBR_NONE if absent
    uint32_t* slot_of;   // [capB] hashtable slot of a brick created by this step's grow
    uint32_t* slist;     // [capB] rows of the bricks that hold new sources (this step's grow work list)
    uint64_t* smask;     // [capB] their source masks
    ulonglong2* table;   // [slots] {brick key, row}
    uint64_t* pend;      // [slots] active bits set in bricks created during the running grow
    uint64_t* bkey2;     // compaction double buffers
    uint64_t* mask2;
    uint64_t* grown2;
    uint32_t* newrow;    // [capB] old row -> new row of the last compaction (NBR_NONE = freed)
    unsigned long long* tile_state;  // scan descriptors
    double* partial;     // block partial sums
};

// The host never swaps pointers: every kernel resolves the double buffers from the device parity
// word, so whole runs can be enqueued without a host round trip per step.
__device__ __forceinline__ Store resolve(const Store& in, const DevState* ds) {
    Store s = in;
    const unsigned par = ds->parity;
    if (par & 1u) { double* t = s.Q; s.Q = s.Qn; s.Qn = t; }
    if (par & 2u) {
        uint64_t* t = s.bkey; s.bkey = s.bkey2; s.bkey2 = t;
        t = s.mask; s.mask = s.mask2; s.mask2 = t;
        t = s.grown; s.grown = s.grown2; s.grown2 = t;
    }
    return s;
}

// ---- key packing (A18): field j at shift (n-1-j)*bits, biased by 2^(bits-1); dim 0 most significant
__device__ __forceinline__ int field_shift(const Params& p, int j) { return (p.n - 1 - j) * p.bits; }

template <int NDIM>
__device__ __forceinline__ void unpack(const Params& p, uint64_t key, int32_t c[NDIM]) {
    const uint64_t m = (1ull << p.bits) - 1ull;
#pragma unroll
    for (int j = 0; j < NDIM; ++j)
        c[j] = (int32_t)((int64_t)((key >> ((NDIM - 1 - j) * p.bits)) & m) - p.bias);
}

template <int NDIM>
__device__ __forceinline__ uint64_t pack(const Params& p, const int32_t c[NDIM]) {
    uint64_t k = 0;
#pragma unroll
    for (int j = 0; j < NDIM; ++j) k |= (uint64_t)((int64_t)c[j] + p.bias) << ((NDIM - 1 - j) * p.bits);
    return k;
}

// ---- hashtable: open addressing, linear probing, 16-byte slots {key, index} --------------------
__device__ __forceinline__ uint64_t mix64(uint64_t x) {  // splitmix64 finaliser
    x ^= x >> 30; x *= 0xbf58476d1ce4e5b9ull;
    x ^= x >> 27; x *= 0x94d049bb133111ebull;
    x ^= x >> 31;
    return x;
}
__device__ __forceinline__ uint64_t home_slot(uint64_t key, uint64_t slots) {
    return __umul64hi(mix64(key), slots);
}

// returns pool index or NBR_NONE. probes (optional) counts slots inspected.
__device__ __forceinline__ uint32_t ht_find(const ulonglong2* __restrict__ table, uint64_t slots,
                                            uint64_t key, unsigned* probes = nullptr) {
    uint64_t s = home_slot(key, slots);
    unsigned np = 0;
    for (;;) {
        const ulonglong2 e = table[s];
        ++np;
        if (e.x == key) { if (probes) *probes += np; return (uint32_t)e.y; }
        if (e.x == KEY_EMPTY) { if (probes) *probes += np; return NBR_NONE; }
        if (++s == slots) s = 0;
    }
}

// Find-or-insert for kernels that mutate the table while others probe it (grow): volatile probes.
// Returns the slot holding `key` (inserted = true if THIS thread claimed it and must publish the
// value), or ~0ull if the table is full.
__device__ __forceinline__ uint64_t ht_upsert(ulonglong2* table, uint64_t slots, uint64_t key, bool& inserted) {
    uint64_t s = home_slot(key, slots);
    inserted = false;
    for (uint64_t tries = 0; tries < slots; ++tries) {
        unsigned long long* kp = reinterpret_cast<unsigned long long*>(&table[s].x);
        unsigned long long cur = *reinterpret_cast<volatile unsigned long long*>(kp);
        if (cur == KEY_EMPTY) {
            cur = atomicCAS(kp, KEY_EMPTY, key);
            if (cur == KEY_EMPTY) { inserted = true; return s; }
        }
        if (cur == key) return s;
        if (++s == slots) s = 0;
    }
    return ~0ull;
}

// Claim a slot for `key` if absent. Returns the slot index if THIS thread inserted (caller then
// publishes the value), or ~0ull if the key was already there / the table is full.
__device__ __forceinline__ uint64_t ht_claim(ulonglong2* table, uint64_t slots, uint64_t key,
                                             unsigned* probes = nullptr) {
    uint64_t s = home_slot(key, slots);
    unsigned np = 0;
    for (uint64_t tries = 0; tries < slots; ++tries) {
        unsigned long long* kp = reinterpret_cast<unsigned long long*>(&table[s].x);
        unsigned long long cur = *reinterpret_cast<volatile unsigned long long*>(kp);
        ++np;
        if (cur == KEY_EMPTY) cur = atomicCAS(kp, KEY_EMPTY, key);
        if (cur == KEY_EMPTY) { if (probes) *probes += np; return s; }
        if (cur == key) { if (probes) *probes += np; return ~0ull; }
        if (++s == slots) s = 0;
    }
    if (probes) *probes += np;
    return ~0ull - 1;  // table full
}

// ---- dynamics (A12): fixed operation order, never fused -------------------------------------
#define DMUL(a, b) __dmul_rn((a), (b))
#define DADD(a, b) __dadd_rn((a), (b))
#define DSUB(a, b) __dsub_rn((a), (b))

// f_j(x) with x[j] replaced by xj (the face coordinate along j)
template <int NDIM, int DYN>
__device__ __forceinline__ double dyn_f(const Params& p, const double x[NDIM], int j, double xj) {
    if constexpr (DYN == 0) {          // Lorenz '63 classic (sigma, beta, rho)
        if (j == 0) return DMUL(p.par[0], DSUB(x[1], xj));
        if (j == 1) return DSUB(DMUL(x[0], DSUB(p.par[2], x[2])), xj);
        return DSUB(DMUL(x[0], x[1]), DMUL(p.par[1], xj));
    } else if constexpr (DYN == 1) {   // Lorenz '63, PAPER.md:303 (sigma, b, r)
        if (j == 0) return DMUL(p.par[0], DSUB(x[1], xj));
        if (j == 1) return DSUB(-xj, DMUL(x[0], x[2]));
        return DSUB(DSUB(DMUL(x[0], x[1]), DMUL(p.par[1], xj)), DMUL(p.par[1], p.par[2]));
    } else if constexpr (DYN == 2) {   // Lorenz '96, PAPER.md:319 (cyclic; x_j itself enters only as -x_j)
        const int jp = (j + 1) % NDIM, jm1 = (j + NDIM - 1) % NDIM, jm2 = (j + NDIM - 2) % NDIM;
        return DADD(DSUB(DMUL(DSUB(x[jp], x[jm2]), x[jm1]), xj), p.par[0]);
    } else if constexpr (DYN == 3) {   // linear, ascending m
        double s = DMUL(p.par[j * NDIM + 0], j == 0 ? xj : x[0]);
#pragma unroll
        for (int m = 1; m < NDIM; ++m) s = DADD(s, DMUL(p.par[j * NDIM + m], m == j ? xj : x[m]));
        return s;
    } else {                           // constant
        return p.par[j];
    }
}

// cell-centre coordinates and the 2n own face velocities of cell c:
//   ul[j] = u_{c,j}   (lower j-face),  uu[j] = u_{c+e^j,j} (upper j-face = lower face of c+e^j)
template <int NDIM, int DYN>
__device__ __forceinline__ void face_velocities(const Params& p, const int32_t c[NDIM],
                                                double ul[NDIM], double uu[NDIM]) {
    double x[NDIM];
#pragma unroll
    for (int m = 0; m < NDIM; ++m) x[m] = DADD(p.mu[m], DMUL((double)c[m], p.h[m]));
#pragma unroll
    for (int j = 0; j < NDIM; ++j) {
        const double xl = DADD(p.mu[j], DMUL((double)c[j] - 0.5, p.h[j]));
        const double xu = DADD(p.mu[j], DMUL((double)c[j] + 0.5, p.h[j]));
        ul[j] = dyn_f<NDIM, DYN>(p, x, j, xl);
        uu[j] = dyn_f<NDIM, DYN>(p, x, j, xu);
    }
}

// the n LOWER face velocities only (all Eq. 8 needs)
template <int NDIM, int DYN>
__device__ __forceinline__ void lower_face_velocities(const Params& p, const int32_t c[NDIM], double ul[NDIM]) {
    double x[NDIM];
#pragma unroll
    for (int m = 0; m < NDIM; ++m) x[m] = DADD(p.mu[m], DMUL((double)c[m], p.h[m]));
#pragma unroll
    for (int j = 0; j < NDIM; ++j) ul[j] = dyn_f<NDIM, DYN>(p, x, j, DADD(p.mu[j], DMUL((double)c[j] - 0.5, p.h[j])));
}

// s_c = sum_j |u_{c,j}| / h_j, ascending j, true division (bit-identical to the oracle's Eq. 8 term)
template <int NDIM>
__device__ __forceinline__ double cfl_term(const Params& p, const double ul[NDIM]) {
    double s = 0.0;
#pragma unroll
    for (int j = 0; j < NDIM; ++j)
        s = DADD(s, p.h_pow2 ? DMUL(fabs(ul[j]), p.hinv[j]) : __ddiv_rn(fabs(ul[j]), p.h[j]));
    return s;
}

// Fold the CFL term of one cell into a running maximum without paying n true divisions per cell:
// s~ = sum_j |u_j| * (1/h_j) differs from the exact term by a few ulp, and only a cell whose s~ comes
// within 1e-12 (relative) of the running maximum can raise it, so the exact term is evaluated for
// those cells only. The maximum that comes out is the exact one, bit for bit.
template <int NDIM>
__device__ __forceinline__ void cfl_fold(const Params& p, const double ul[NDIM], double& best) {
    double sa = 0.0;
#pragma unroll
    for (int j = 0; j < NDIM; ++j) sa = fma(fabs(ul[j]), p.hinv[j], sa);
    if (sa >= best * (1.0 - 1e-12)) best = fmax(best, cfl_term<NDIM>(p, ul));
}

// active table size for NB bricks: room for the brick count to grow 8x before the load factor is
// reached, never below 2^16 slots, never above the allocation
__host__ __device__ __forceinline__ unsigned long long table_slots_for(const Params& p, unsigned long long NB) {
    unsigned long long want = (unsigned long long)((double)NB * 8.0 / p.load_factor) + 1ull;
    if (want < (1ull << 16)) want = 1ull << 16;
    return want < p.slots ? want : p.slots;
}

// monotonised-central limiter, division-free (A3)
__device__ __forceinline__ double mc_limit(double a, double b) {
    if (a * b <= 0.0) return 0.0;
    const double m = fmin(0.5 * fabs(a + b), fmin(2.0 * fabs(a), 2.0 * fabs(b)));
    return a > 0.0 ? m : -m;
}

// same limiter, cheaper: sign test on the high words instead of a product (differs from mc_limit only
// when a*b underflows to zero, where the result is below 1e-150 anyway)
// (plain compare-and-select minimum: the operands are never NaN, and fmin's NaN handling costs ~8
// instructions per call in SASS)
__device__ __forceinline__ double dmin(double a, double b) { return a < b ? a : b; }
__device__ __forceinline__ double mc_limit_fast(double a, double b) {
    if ((__double2hiint(a) ^ __double2hiint(b)) < 0) return 0.0;
    const double fa = fabs(a), fb = fabs(b);
    const double m1 = dmin(fa, fb);
    const double m = dmin(0.5 * (fa + fb), m1 + m1);      // same sign: |a + b| = |a| + |b|
    return copysign(m, a);
}

}  // namespace gbees
