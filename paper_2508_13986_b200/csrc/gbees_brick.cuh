// Kernels of the GBEES prediction step on the dense-brick store.
// Every phase is a grid-stride __device__ function, so the same code runs as a stream of launches
// (gbees_step / gbees_prune / gbees_run) or inside the persistent single-cluster loop for small
// grids (k_run_small). Semantics: DESIGN.md D1-D5 (= SURVEY.md 8(c)).
//
// Brick geometry: 64 cell slots per brick, 2^K_j cells along dimension j (sum K_j = 6; n = 6: a
// 2x2x2x2x2x2 box). Local index l = concatenation of the low K_j bits of every coordinate, dim 0
// most significant. One warp works on one brick; neighbour values inside the brick come from
// shared memory, values across a brick face from the neighbour brick's row (coalesced 8-byte loads
// of a contiguous 512-byte row), so the per-cell adjacency and per-cell keys of a cell list are gone.
#pragma once
#include <cuda_pipeline.h>
#include "gbees_prims.cuh"

namespace gbees {

constexpr int WPB = TPB / 32;   // warps (= bricks in flight) per block

template <int NDIM>
struct Geo {
    __host__ __device__ static constexpr int K(int j) { return 6 / NDIM + (j < 6 % NDIM ? 1 : 0); }
    __host__ __device__ static constexpr int SH(int j) {
        int s = 0;
        for (int m = j + 1; m < NDIM; ++m) s += K(m);
        return s;
    }
    __host__ __device__ static constexpr int MK(int j) { return (1 << K(j)) - 1; }
    // index of local cell l on a j-face (the bits of dimension j removed)
    __host__ __device__ static constexpr int fidx(int j, int l) {
        return ((l >> (SH(j) + K(j))) << SH(j)) | (l & ((1 << SH(j)) - 1));
    }
};

__device__ __forceinline__ unsigned gwarp() { return (blockIdx.x * blockDim.x + threadIdx.x) >> 5; }
__device__ __forceinline__ unsigned gwarps() { return (gridDim.x * blockDim.x) >> 5; }
__device__ __forceinline__ unsigned lane_id() { return threadIdx.x & 31; }

// cell coordinates of local slot l in the brick with coordinates B
template <int NDIM>
__device__ __forceinline__ void cell_coords(const int32_t B[NDIM], int l, int32_t c[NDIM]) {
#pragma unroll
    for (int j = 0; j < NDIM; ++j) c[j] = B[j] * (1 << Geo<NDIM>::K(j)) + ((l >> Geo<NDIM>::SH(j)) & Geo<NDIM>::MK(j));
}
// brick coordinates + local slot of cell c
template <int NDIM>
__device__ __forceinline__ int cell_to_brick(const int32_t c[NDIM], int32_t B[NDIM]) {
    int l = 0;
#pragma unroll
    for (int j = 0; j < NDIM; ++j) {
        B[j] = c[j] >> Geo<NDIM>::K(j);                         // arithmetic shift = floor
        l |= (c[j] & Geo<NDIM>::MK(j)) << Geo<NDIM>::SH(j);
    }
    return l;
}

// dt of Eq. (8) with the caller's cap (every thread computes the same value)
__device__ __forceinline__ double step_dt(const Params& p, const DevState* ds) {
    const double smax = __longlong_as_double((long long)ds->smax_bits);
    const double cap = ds->dt_cap;
    const bool capped = isfinite(cap) && cap > 0.0;
    double dt = smax > 0.0 ? __ddiv_rn(p.cfl, smax) : (capped ? cap : 0.0);
    if (capped && cap < dt) dt = cap;
    return dt;
}

// ---- a1 grow / a7 mark: Targets(c), D1.1 / A10 / A11 -------------------------------------------
// Targets are numbered t in [0, 2n + 4 C(n,2)): t < 2n is the face target (dim t>>1, side t&1);
// the rest are edge targets (pair (j<l), side_j, side_l).
template <int NDIM>
__device__ __forceinline__ void decode_target(int t, int& j, int& sj, int& l, int& sl) {
    if (t < 2 * NDIM) { j = t >> 1; sj = t & 1; l = -1; sl = 0; return; }
    int e = t - 2 * NDIM;
    sl = e & 1; sj = (e >> 1) & 1;
    int pair = e >> 2;           // pairs in order (0,1),(0,2),...,(0,n-1),(1,2),...
    j = 0;
    int row = NDIM - 1;
    while (pair >= row) { pair -= row; --row; ++j; }
    l = j + 1 + pair;
}

// GROW = true  (Alg. 2 without staging: atomicCAS claims the brick slot):
//   sources = active cells with P >= p* whose targets were not inserted yet; every target cell is
//   activated (bit set in its brick's mask; the brick is created if absent).
// GROW = false (Alg. 3 line "mark"): sources = all cells with P >= p*; the source and
//   every existing target get a keep mark.
// Bit-parallel per brick: one warp turns the sources' outflow flags into 2n slot masks O_d, then
// every lane takes target classes t (a face step or a pair of steps), ANDs the masks of the steps
// involved, shifts the result to the target slots and splits it by destination brick (own, face
// neighbour, diagonal). Masks bound for the own brick and the 2n face neighbours are merged with
// warp OR-reductions, so a brick costs O(2n + diagonals) global atomics instead of O(cells x targets).
template <int NDIM>
__device__ __forceinline__ unsigned long long edge_mask(int j, int side) {   // slots whose step (j, side) leaves the brick
    unsigned long long e = 0ull;
    const int SH = Geo<NDIM>::SH(j), MK = Geo<NDIM>::MK(j);
    for (int l = 0; l < 64; ++l)
        if (((l >> SH) & MK) == (side ? MK : 0)) e |= 1ull << l;
    return e;
}

// GROW: activate the cells `bits` of the brick in row `row` (NBR_NONE: unknown, look `key` up and create it if
// absent). Returns the bits this thread switched on: the CFL terms are folded for the NEW cells only (folding them
// for every target, so that the atomics need not return, was measured: 5-20 % slower on both small and large grids).
__device__ __forceinline__ unsigned long long grow_apply(const Params& p, const Store& st, DevState* ds, uint32_t NB0,
                                                               uint64_t slots, int nd, uint32_t row, uint64_t key,
                                                               unsigned long long bits) {
    if (row == NBR_NONE) {
        bool inserted;
        const uint64_t s = ht_upsert(st.table, slots, key, inserted);
        if (s == ~0ull) { atomicOr(&ds->err, E_TABLE_FULL); return 0ull; }
        if (inserted) {
            const uint32_t nr = atomicAdd(&ds->NB, 1u);
            if (nr >= p.capB) { atomicOr(&ds->err, E_CAPACITY); return 0ull; }
            st.bkey[nr] = key; st.slot_of[nr] = (uint32_t)s; st.grown[nr] = 0ull; st.mask[nr] = 0ull;
            for (int d = 0; d < nd; ++d) st.adj[(size_t)nr * nd + d] = NBR_NONE;
            __threadfence();
            *reinterpret_cast<volatile unsigned long long*>(&st.table[s].y) = nr;
        } else {
            const uint32_t er = (uint32_t)*reinterpret_cast<volatile unsigned long long*>(&st.table[s].y);
            if (er != NBR_NONE && er < NB0) row = er;
        }
        if (row == NBR_NONE) return bits & ~atomicOr((unsigned long long*)&st.pend[s], bits);
    }
    // (most target cells exist already: the plain read saves the atomic, which would serialise in L2)
    const unsigned long long want = bits & ~*reinterpret_cast<volatile unsigned long long*>(&st.mask[row]);
    if (!want) return 0ull;
    return want & ~atomicOr((unsigned long long*)&st.mask[row], want);
}

// a1, first half: list the bricks that hold NEW sources (active, P >= p*, targets not inserted yet) with
// their source masks. The expensive half (phase_targets) then runs over that list, evenly spread over the
// warps; here a brick costs two dependent loads. A cell grows once (autonomous f): its GROWN bit is set here.
__device__ inline void phase_detect(const Params& p, const Store& st, DevState* ds) {
    const uint32_t NB0 = ds->NB_before_grow;
    const double scale = ds->scale;
    const unsigned lane = lane_id();
    for (uint32_t b = gwarp(); b < NB0; b += gwarps()) {   // warp-uniform
        const uint64_t m = st.mask[b], g = st.grown[b];
        const uint64_t cand = m & ~g;
        if (!cand) continue;
        const bool s0 = ((cand >> lane) & 1ull) && scale * st.Q[(size_t)b * 64 + lane] >= p.thresh;
        const bool s1 = ((cand >> (lane + 32)) & 1ull) && scale * st.Q[(size_t)b * 64 + 32 + lane] >= p.thresh;
        const uint64_t src = (uint64_t)__ballot_sync(0xffffffffu, s0) | ((uint64_t)__ballot_sync(0xffffffffu, s1) << 32);
        if (!src || lane != 0) continue;
        const uint32_t i = atomicAdd(&ds->nsrc, 1u);
        st.slist[i] = b;
        st.smask[i] = src;
        st.grown[b] = g | src;
    }
}

// SKIP: a class iteration in which no lane has a part is skipped. That pays when the pass is throughput-bound (mark;
// grow on large grids); without the branch the three iterations overlap, which pays when one warp's latency is the
// bound (grow on small grids: a few thousand listed bricks, one warp each).
template <int NDIM, int DYN, bool GROW, bool SKIP = true>
__device__ void phase_targets(const Params& p, const Store& st, DevState* ds) {
    using G = Geo<NDIM>;
    constexpr int ND = 2 * NDIM, NT = ND + 2 * NDIM * (NDIM - 1), OWN = ND;
    __shared__ unsigned long long sO[WPB][ND];        // O_d: sources with outflow through face d
    __shared__ unsigned long long sDiag[WPB][NT - ND > 0 ? NT - ND : 1];   // target bits bound for diagonal bricks, per edge class
    __shared__ uint32_t sAdj[WPB][ND];
    __shared__ unsigned long long sTb[WPB][ND + 1];   // merged target bits per destination (face neighbours, own)
    __shared__ uint8_t sItem[WPB][NT + 1];            // work list of the non-empty destinations / diagonal classes
    __shared__ unsigned long long sEdge[ND];
    // new cells: (brick key, bits); one entry per work item at most (own brick + 2n faces + NT - 2n diagonal classes)
    __shared__ unsigned long long sQk[GROW ? WPB : 1][GROW ? NT + 1 : 1], sQm[GROW ? WPB : 1][GROW ? NT + 1 : 1];
    __shared__ unsigned sQn[WPB];
    __shared__ unsigned sQo[GROW ? WPB : 1][GROW ? NT + 1 : 1];   // exclusive prefix of the new-cell counts
    if (threadIdx.x < ND) sEdge[threadIdx.x] = edge_mask<NDIM>(threadIdx.x >> 1, threadIdx.x & 1);
    __syncthreads();
    const uint32_t NB0 = GROW ? ds->NB_before_grow : min(ds->NB, p.capB);
    const double scale = ds->scale;
    const uint64_t slots = ds->slots;
    const int32_t lo = (int32_t)(-p.bias), hi = (int32_t)(p.bias - 1);
    const unsigned w = threadIdx.x >> 5, lane = lane_id();
    const double smax0 = GROW ? __longlong_as_double((long long)ds->smax_bits) : 0.0;   // the maximum so far: most new cells stay below it
    double smax = smax0;
    // new cells (GROW) are queued per warp as (brick key, bits) and expanded by all lanes below
    auto account = [&](uint64_t key, unsigned long long bits) {
        const unsigned k = atomicAdd(&sQn[GROW ? w : 0], 1u);
        sQk[GROW ? w : 0][GROW ? k : 0] = key;
        sQm[GROW ? w : 0][GROW ? k : 0] = bits;
    };
    // GROW: the bricks that hold new sources were listed by phase_detect, so every warp gets the same share of
    // the expensive bricks; mark: all bricks, sources = every cell with P >= p*.
    const uint32_t nwork = GROW ? min(ds->nsrc, p.capB) : NB0;
    for (uint32_t wi = gwarp(); wi < nwork; wi += gwarps()) {   // warp-uniform
        const uint32_t b = GROW ? st.slist[wi] : wi;
        const uint64_t m = st.mask[b];
        const uint64_t bk = st.bkey[b];
        const uint32_t my_adj = lane < ND ? st.adj[(size_t)b * ND + lane] : NBR_NONE;
        const uint64_t cand = GROW ? st.smask[wi] : m;        // GROW: the sources themselves
        if (!cand) continue;
        int32_t B[NDIM];
        unpack<NDIM>(p, bk, B);
        unsigned fl[2] = {0u, 0u};
        uint64_t src = 0;
#pragma unroll
        for (int hh = 0; hh < 2; ++hh) {
            const int l = (int)lane + 32 * hh;
            bool is_src = false;
            if ((cand >> l) & 1ull) is_src = GROW ? true : scale * st.Q[(size_t)b * 64 + l] >= p.thresh;
            if (is_src) {
                int32_t c[NDIM];
                cell_coords<NDIM>(B, l, c);
                double ul[NDIM], uu[NDIM];
                face_velocities<NDIM, DYN>(p, c, ul, uu);
                unsigned f = 0, border = 0;
#pragma unroll
                for (int j = 0; j < NDIM; ++j) {
                    f |= (ul[j] < 0.0 ? 1u : 0u) << (2 * j);
                    f |= (uu[j] > 0.0 ? 1u : 0u) << (2 * j + 1);
                    border |= (c[j] <= lo ? 1u : 0u) << (2 * j);
                    border |= (c[j] >= hi ? 1u : 0u) << (2 * j + 1);
                }
                if (f & border) {                        // a target would leave the packable range (A18)
                    if (GROW) atomicOr(&ds->err, E_KEY_RANGE);
                    f &= ~border;
                }
                fl[hh] = f;
            }
            src |= (uint64_t)__ballot_sync(0xffffffffu, is_src) << (32 * hh);
        }
        if (!src) continue;
        if (lane < ND) sAdj[w][lane] = my_adj;
        if (lane == 0) sQn[w] = 0u;
#pragma unroll
        for (int d = 0; d < ND; ++d) {
            const unsigned long long od = (unsigned long long)__ballot_sync(0xffffffffu, (fl[0] >> d) & 1u) |
                                          ((unsigned long long)__ballot_sync(0xffffffffu, (fl[1] >> d) & 1u) << 32);
            if (lane == 0) sO[w][d] = od;
        }
        __syncwarp();
        // ---- target classes: shift the source masks to the target slots, split by destination brick.
        // No atomics here: the parts bound for the own brick and the 2n face neighbours are merged
        // across the lanes with warp OR-reductions (lane d keeps destination d); a diagonal part is
        // parked in shared memory under its class number.
        unsigned long long myT = (!GROW && lane == OWN) ? src : 0ull;   // mark: sources keep themselves
#pragma unroll
        for (int it = 0; it < (NT + 31) / 32; ++it) {
            const int t = (int)lane + 32 * it;
            unsigned long long vOwn = 0ull, v1 = 0ull, v2 = 0ull;
            int d1 = -1, d2 = -1;
            if (t < NT) {
                int j, sj, l2, sl;
                decode_target<NDIM>(t, j, sj, l2, sl);
                d1 = 2 * j + sj;
                unsigned long long S = sO[w][d1];
                if (l2 >= 0) S &= sO[w][2 * l2 + sl];
                const int s1 = 1 << G::SH(j), w1 = G::MK(j) * s1;
                unsigned long long in = S & ~sEdge[d1], cr = S & sEdge[d1];     // stay in the brick / cross face d1
                in = sj ? in << s1 : in >> s1;
                cr = sj ? cr >> w1 : cr << w1;
                if (l2 < 0) { vOwn = in; v1 = cr; }
                else {
                    d2 = 2 * l2 + sl;
                    const int s2 = 1 << G::SH(l2), w2 = G::MK(l2) * s2;
                    const unsigned long long e2 = sEdge[d2];
                    unsigned long long p00 = in & ~e2, p01 = in & e2, p10 = cr & ~e2, p11 = cr & e2;
                    vOwn = sl ? p00 << s2 : p00 >> s2;
                    v1 = sl ? p10 << s2 : p10 >> s2;
                    v2 = sl ? p01 >> w2 : p01 << w2;
                    sDiag[w][t - ND] = sl ? p11 >> w2 : p11 << w2;
                }
            }
            if (SKIP && !__any_sync(0xffffffffu, (vOwn | v1 | v2) != 0ull)) continue;
#pragma unroll
            for (int d = 0; d <= ND; ++d) {
                const unsigned long long x = d == OWN ? vOwn : ((d == d1 ? v1 : 0ull) | (d == d2 ? v2 : 0ull));
                const unsigned lo32 = __reduce_or_sync(0xffffffffu, (unsigned)x);
                const unsigned hi32 = __reduce_or_sync(0xffffffffu, (unsigned)(x >> 32));
                if ((int)lane == d) myT |= ((unsigned long long)hi32 << 32) | lo32;
            }
        }
        __syncwarp();
        // ---- apply: the non-empty parts (2n + 1 merged destinations, up to 4 C(n,2) diagonal classes)
        // are compacted into one work list, so that all of them go through their chain of dependent
        // global operations (adjacency, mask, atomic) at the same time, one lane per item
        if (lane <= ND) sTb[w][lane] = myT;
        unsigned nitems = 0;
        {
            const unsigned bal = __ballot_sync(0xffffffffu, lane <= ND && myT != 0ull);
            if (lane <= ND && myT) sItem[w][__popc(bal & ((1u << lane) - 1u))] = (uint8_t)lane;
            nitems = __popc(bal);
#pragma unroll
            for (int it = 0; it < (NT - ND + 31) / 32; ++it) {
                const int t = ND + (int)lane + 32 * it;
                const bool nz = t < NT && sDiag[w][t - ND] != 0ull;
                const unsigned bl = __ballot_sync(0xffffffffu, nz);
                if (nz) sItem[w][nitems + __popc(bl & ((1u << lane) - 1u))] = (uint8_t)(t + 1);   // ND + 1 .. NT: class t
                nitems += __popc(bl);
            }
        }
        __syncwarp();
        for (unsigned it = lane; it < nitems; it += 32) {
            const int code = sItem[w][it];
            uint32_t row;
            uint64_t key = bk;
            unsigned long long bits;
            if (code <= ND) {                        // own brick or face neighbour code
                bits = sTb[w][code];
                row = code == OWN ? b : sAdj[w][code];
                if (code != OWN) {
                    const uint64_t u1 = 1ull << ((NDIM - 1 - (code >> 1)) * p.bits);
                    key = (code & 1) ? bk + u1 : bk - u1;
                }
            } else {                                 // diagonal brick of edge class t = code - 1
                const int t = code - 1;
                bits = sDiag[w][t - ND];
                int j, sj, l2, sl;
                decode_target<NDIM>(t, j, sj, l2, sl);
                const int d1 = 2 * j + sj, d2 = 2 * l2 + sl;
                // through the adjacency of either face neighbour, else by key
                row = NBR_NONE;
                const uint32_t r1 = sAdj[w][d1], r2 = sAdj[w][d2];
                if (r1 != NBR_NONE) row = st.adj[(size_t)r1 * ND + d2];
                if (row == NBR_NONE && r2 != NBR_NONE) row = st.adj[(size_t)r2 * ND + d1];
                const uint64_t u1 = 1ull << ((NDIM - 1 - j) * p.bits), u2 = 1ull << ((NDIM - 1 - l2) * p.bits);
                key = sj ? bk + u1 : bk - u1;
                key = sl ? key + u2 : key - u2;
                if (!GROW && row == NBR_NONE) row = ht_find(st.table, slots, key);
            }
            if (GROW) {
                const unsigned long long fresh = grow_apply(p, st, ds, NB0, slots, ND, row, key, bits);
                if (fresh) account(key, fresh);
            } else if (row != NBR_NONE) {
                const unsigned long long x = bits & st.mask[row];
                if (x) atomicOr((unsigned long long*)&st.keep[row], x);
            }
        }
        __syncwarp();
        if (GROW) {   // fold the CFL terms of the new cells into the running maximum (Eq. 8):
            // the queued (brick, bits) pairs are flattened so that every lane takes one cell at a time
            const unsigned nq = sQn[w];
            if (nq) {
                unsigned run = 0;
                for (unsigned base = 0; base < nq; base += 32) {
                    const unsigned k = base + lane;
                    const unsigned cnt = k < nq ? (unsigned)__popcll(sQm[w][k]) : 0u;
                    unsigned inc = cnt;
#pragma unroll
                    for (int o = 1; o < 32; o <<= 1) {
                        const unsigned v = __shfl_up_sync(0xffffffffu, inc, o);
                        if ((int)lane >= o) inc += v;
                    }
                    if (k < nq) sQo[w][k] = run + inc - cnt;
                    run += __shfl_sync(0xffffffffu, inc, 31);
                }
                __syncwarp();
                for (unsigned idx = lane; idx < run; idx += 32) {
                    unsigned k = 0;
                    while (k + 1 < nq && sQo[w][k + 1] <= idx) ++k;
                    unsigned r = idx - sQo[w][k];
                    unsigned long long mm = sQm[w][k];
                    while (r--) mm &= mm - 1ull;
                    const int tl = __ffsll((long long)mm) - 1;
                    int32_t TB[NDIM], tc[NDIM];
                    unpack<NDIM>(p, sQk[w][k], TB);
                    cell_coords<NDIM>(TB, tl, tc);
                    double ul[NDIM];
                    lower_face_velocities<NDIM, DYN>(p, tc, ul);
                    cfl_fold<NDIM>(p, ul, smax);
                }
                __syncwarp();
            }
        }
    }
    if (GROW) {
        smax = block_max(smax);
        if (threadIdx.x == 0 && smax > smax0) atomicMax(&ds->smax_bits, (unsigned long long)__double_as_longlong(smax));
    }
}

// ---- brick adjacency (here per brick instead of per cell) -------------------------
// ALL = true: every brick (after init / import / prune); false: the bricks created by this step's
// grow, which also take their active bits from pend[] and patch their neighbours' rows.
template <int NDIM, bool ALL>
__device__ void phase_link(const Params& p, const Store& st, DevState* ds) {
    constexpr int ND = 2 * NDIM;
    const uint32_t first = ALL ? 0u : ds->NB_before_grow;
    const uint32_t NB = min(ds->NB, p.capB);
    const uint64_t slots = ds->slots;
    const uint64_t items = (uint64_t)(NB - first) * ND;
    const uint64_t fmask = (1ull << p.bits) - 1ull;
    for (uint64_t w = gtid(); w < items; w += gthreads()) {
        const uint32_t row = first + (uint32_t)(w / ND);
        const int d = (int)(w % ND), j = d >> 1;
        const uint64_t key = st.bkey[row];
        const int fs = (NDIM - 1 - j) * p.bits;
        const uint64_t fld = (key >> fs) & fmask;
        uint32_t nb = NBR_NONE;
        if ((d & 1) ? (fld != fmask) : (fld != 0)) nb = ht_find(st.table, slots, (d & 1) ? key + (1ull << fs) : key - (1ull << fs));
        st.adj[(size_t)row * ND + d] = nb;
        if (!ALL) {
            if (nb != NBR_NONE) st.adj[(size_t)nb * ND + (d ^ 1)] = row;
            if (d == 0) {
                const uint32_t s = st.slot_of[row];
                st.mask[row] = st.pend[s];
                st.pend[s] = 0ull;
            }
        }
    }
}

// CFL maximum over all active cells (init / import / after a prune; grow maintains it incrementally)
template <int NDIM, int DYN>
__device__ void phase_smax(const Params& p, const Store& st, DevState* ds) {
    const uint32_t NB = min(ds->NB, p.capB);
    const uint64_t items = (uint64_t)NB * 64;
    double smax = 0.0;
    for (uint64_t i = gtid(); i < items; i += gthreads()) {
        const uint32_t b = (uint32_t)(i >> 6);
        const int l = (int)(i & 63);
        if (!((st.mask[b] >> l) & 1ull)) continue;
        int32_t B[NDIM], c[NDIM];
        unpack<NDIM>(p, st.bkey[b], B);
        cell_coords<NDIM>(B, l, c);
        double ul[NDIM];
        lower_face_velocities<NDIM, DYN>(p, c, ul);
        cfl_fold<NDIM>(p, ul, smax);
    }
    smax = block_max(smax);
    if (threadIdx.x == 0 && smax > 0.0) atomicMax(&ds->smax_bits, (unsigned long long)__double_as_longlong(smax));
}

// ---- a2+a4 pass 1: every active cell computes the fluxes of the faces it is UPWIND of -----------
// Gather form D2 (= Eq. 7 + Alg. 1 + high-resolution term), written in
// Courant numbers a = tau_j u (tau_j = dt / h_j), so that every quantity below is tau_j * flux:
//   T_l   = 1/2 [ a+_{c,l} (P_c - P_{c-e^l}) + a-_{c+e^l,l} (P_{c+e^l} - P_c) ]
//   G_j   = P*_{c,(j)} = P_c - sum_{l != j} T_l
//   sig_j = mc(P_c - P_{c-e^j}, P_{c+e^j} - P_c)     (limited wave when c is the upwind cell)
//   upper face, a = a_{c+e^j,j} > 0:  F = a (G_j + 1/2 (1 - a) sig_j)
//   lower face, a = a_{c,j}     < 0:  F = a (G_j - 1/2 (1 + a) sig_j)
// A face whose upwind cell is NOT active carries only the high-resolution term; the active downwind
// cell computes it (needs the two-hop value) and keeps it to itself.
// F goes to both cells of the face: inside the brick through the face array Fb (written by the one
// upwind owner, applied to both sides after the cell loop), across a brick face the owner applies it to
// itself and leaves it in phi[] (the downwind cell sets its fetch bit and picks it up in pass 2).
// Qn <- P_c - sum_j (F_up - F_lo) over the faces resolved inside the brick.
//
// Face velocities. Every dynamics id is affine in x_j for fixed other coordinates:
// f_j(x) = A_j(x_{!=j}) + B_j x_j, so a_lo = tau_j A_j + (tau_j B_j) x_lo and a_up likewise with x_up:
// one evaluation of A_j serves both faces, and the two cells of a face compute the same bits for its
// Courant number (same A_j, same table entry for the face coordinate), which is what keeps "who is
// upwind" consistent between them. The coordinates come from a per-brick table (2^K_j centres and
// 2^K_j + 1 faces per dimension, A12 arithmetic). These Courant numbers serve the fluxes only; grow,
// prune and dt use the unfused A12 velocities of gbees_common.cuh.
template <int NDIM>
struct FluxGeo {
    using G = Geo<NDIM>;
    __host__ __device__ static constexpr int XC(int j) { int o = 0; for (int m = 0; m < j; ++m) o += 1 << G::K(m); return o; }
    __host__ __device__ static constexpr int XF(int j) { return XC(j) + j; }
    static constexpr int NC = XC(NDIM), NF = XC(NDIM) + NDIM;
    // face array: one entry per in-brick face and dimension, addressed by the slot of the face's LOWER cell
    // (64 entries per dimension; packing them to the 32 that a two-cell-wide dimension uses costs more index
    // arithmetic per cell than the shared memory is worth while registers cap the occupancy at 2 blocks per SM)
    // every dimension two cells wide (n = 6): only HALF of each neighbour row is ever read -- the cells that face
    // this brick -- so the two neighbour rows of a dimension are staged as ONE combined row (see Flux1Smem::R)
    __host__ __device__ static constexpr bool all_two() { for (int j = 0; j < NDIM; ++j) if (G::K(j) != 1) return false; return true; }
    static constexpr bool ALL2 = all_two();
    // (ALL2: a dimension has 32 in-brick faces, entered under the slot of the lower cell with bit j removed)
    static constexpr int FB = ALL2 ? 32 : 64;
    __host__ __device__ static constexpr int fb(int j, int l) { return ALL2 ? G::fidx(j, l) : l; }
};

// Shared memory of one warp in pass 1
template <int NDIM>
struct alignas(16) Flux1Smem {
    // staged rows. General geometry: the 2n neighbour bricks' rows (index d = 2j + side), then the brick's own row.
    // ALL2 geometry: one combined row per dimension j -- slot l' holds the value of the cell at slot l' of the
    // LOWER neighbour brick if bit j of l' is set (it is the lower neighbour of the own cell l' ^ s), of the UPPER
    // neighbour brick if the bit is clear (the upper neighbour of l' ^ s) -- then the own row: n + 1 rows, not 2n + 1.
    static constexpr bool ALL2 = FluxGeo<NDIM>::ALL2;
    static constexpr int ROWS = ALL2 ? NDIM + 1 : 2 * NDIM + 1, OWN = ROWS - 1;
    double R[ROWS][64];
    double Fb[NDIM][FluxGeo<NDIM>::FB];   // F through the UPPER j-face of slot l, faces inside the brick only
    double acc[64];                  // P_c minus / plus the fluxes the cell applied to itself
    double xc[FluxGeo<NDIM>::NC];    // cell-centre coordinates per dimension and local index
    double xf[FluxGeo<NDIM>::NF];    // face coordinates: entry i = lower face of local index i
    unsigned long long A[2 * NDIM];  // bit l of A[d]: the neighbour of slot l in direction d is active
    unsigned long long RZ[2 * NDIM]; // bit l of RZ[d]: slot l active, that neighbour NOT active, the cell behind it active
    uint32_t adjr[2 * NDIM];         // rows of the 2n neighbour bricks (ALL2: two-hop values are read from global memory)
    uint16_t fl[64];
};
// Shared memory of one warp in pass 1: NBW bricks in flight and their common cell list ((brick << 6) | slot)
template <int NDIM>
struct alignas(16) Flux1Warp {
    static constexpr int NBW = FluxGeo<NDIM>::ALL2 ? 2 : 1;
    Flux1Smem<NDIM> b[NBW];
    uint8_t list[64 * NBW];
};

// A_j and B_j of f_j = A_j + B_j x_j (operation order fixed by the explicit intrinsics)
template <int NDIM, int DYN>
__device__ __forceinline__ double dyn_A(const Params& p, const double x[NDIM], int j) {
    if constexpr (DYN == 0) {
        if (j == 0) return DMUL(p.par[0], x[1]);
        if (j == 1) return DMUL(x[0], DSUB(p.par[2], x[2]));
        return DMUL(x[0], x[1]);
    } else if constexpr (DYN == 1) {
        if (j == 0) return DMUL(p.par[0], x[1]);
        if (j == 1) return -DMUL(x[0], x[2]);
        return __fma_rn(x[0], x[1], -DMUL(p.par[1], p.par[2]));
    } else if constexpr (DYN == 2) {
        const int jp = (j + 1) % NDIM, jm1 = (j + NDIM - 1) % NDIM, jm2 = (j + NDIM - 2) % NDIM;
        return __fma_rn(DSUB(x[jp], x[jm2]), x[jm1], p.par[0]);
    } else if constexpr (DYN == 3) {
        double s = 0.0;
#pragma unroll
        for (int m = 0; m < NDIM; ++m) if (m != j) s = __fma_rn(p.par[j * NDIM + m], x[m], s);
        return s;
    } else {
        return p.par[j];
    }
}
template <int NDIM, int DYN>
__device__ __forceinline__ double dyn_B(const Params& p, int j) {
    if constexpr (DYN == 0) return j == 0 ? -p.par[0] : (j == 1 ? -1.0 : -p.par[1]);
    else if constexpr (DYN == 1) return j == 0 ? -p.par[0] : (j == 1 ? -1.0 : -p.par[1]);
    else if constexpr (DYN == 2) return -1.0;
    else if constexpr (DYN == 3) return p.par[j * NDIM + j];
    else return 0.0;
}

// sign tests on the high word (a value below 2^-1022 in magnitude counts as zero: its flux is zero anyway)
__device__ __forceinline__ bool dpos(double a) { return __double2hiint(a) > 0; }
__device__ __forceinline__ bool dneg(double a) { return __double2hiint(a) < 0; }

// FAST = true: production setting (hi_res on, MC limiter) compiled in; false: flags read at run time
template <int NDIM, int DYN, bool FAST>
__device__ void phase_flux1(const Params& p, const Store& st, DevState* ds) {
    using G = Geo<NDIM>;
    using FG = FluxGeo<NDIM>;
    using SM = Flux1Smem<NDIM>;
    constexpr int ND = 2 * NDIM, OWN = SM::OWN, LOWN = ND;   // OWN: staged row of the brick itself; LOWN: the lane that holds its row / mask
    constexpr bool ALL2 = SM::ALL2;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const unsigned w = threadIdx.x >> 5, lane = lane_id();
    constexpr int NBW = Flux1Warp<NDIM>::NBW;
    Flux1Warp<NDIM>& ws = reinterpret_cast<Flux1Warp<NDIM>*>(smem_raw)[w];
    SM* const smw = ws.b;
    uint8_t* const wlist = ws.list;
    const uint32_t NB = min(ds->NB, p.capB);
    const double dt = step_dt(p, ds);
    const bool hires = FAST || p.hi_res != 0, nolim = !FAST && p.limiter != 0;
    const double* __restrict__ Q = st.Q;
    double tau[NDIM], tauB[NDIM];
#pragma unroll
    for (int j = 0; j < NDIM; ++j) { tau[j] = dt / p.h[j]; tauB[j] = __dmul_rn(tau[j], (dyn_B<NDIM, DYN>(p, j))); }
    // lane d < 2n builds the neighbour-activity masks of direction d: its geometry, once.
    //   edge / w : slots whose step in direction d leaves the brick, and the shift that wraps them into the neighbour
    //   edge2 / w2: the same for a step of two cells
    unsigned long long my_edge = 0ull, my_edge2 = 0ull;
    int my_s = 0, my_w = 0, my_w2 = 0;
    if (lane < ND) {
        const int j = lane >> 1, side = lane & 1;
        my_edge = edge_mask<NDIM>(j, side);
#pragma unroll
        for (int m = 0; m < NDIM; ++m)
            if (m == j) {
                my_s = 1 << G::SH(m); my_w = G::MK(m) << G::SH(m); my_w2 = (G::MK(m) - 1) << G::SH(m);
                for (int l = 0; l < 64; ++l) {
                    const int lj = (l >> G::SH(m)) & G::MK(m);
                    if (side ? lj + 2 > G::MK(m) : lj < 2) my_edge2 |= 1ull << l;
                }
            }
    }
    constexpr uint32_t zrow = NBR_NONE;                     // missing neighbour brick: its staged row is zero-filled
    const uint64_t qlane = reinterpret_cast<uint64_t>(Q) + 16ull * lane;
    // A warp works on NBW bricks at a time: their active cells go into ONE list that is worked off 32 cells at a
    // time, whichever brick a cell belongs to (a brick holds 20-38 active cells: one brick at a time leaves 25-45 %
    // of the lanes of its last iteration idle). Two bricks fit in shared memory only with the combined rows.
    // Metadata of the warp's next NBW bricks is loaded one round ahead.
    uint32_t nx_row[NBW];
    uint64_t nx_mask[NBW], nx_bk[NBW];
    auto fetch_rows = [&](uint32_t b0) {   // (nothing here may USE what it loads: the loads stay in flight behind the cell loop)
#pragma unroll
        for (int u = 0; u < NBW; ++u) {
            const uint32_t bb = b0 + u * gwarps();
            nx_row[u] = zrow; nx_bk[u] = 0ull;
            if (bb < NB) {
                if (lane < ND) nx_row[u] = st.adj[(size_t)bb * ND + lane];     // NBR_NONE = zrow: a missing neighbour
                else if (lane == LOWN) nx_row[u] = bb;
                nx_bk[u] = st.bkey[bb];
            }
        }
    };
    auto fetch_masks = [&]() {
#pragma unroll
        for (int u = 0; u < NBW; ++u) nx_mask[u] = (lane <= LOWN && nx_row[u] != zrow) ? st.mask[nx_row[u]] : 0ull;
    };
    fetch_rows(gwarp());
    fetch_masks();
    unsigned ncells = 0;                                    // active cells of this warp's bricks (the grow does not count)
    for (uint32_t b0 = gwarp(); b0 < NB; b0 += NBW * gwarps()) {   // warp-uniform
        uint64_t mu[NBW];                                   // active masks of the round's bricks (0: no such brick)
        int cbase[NBW + 1];                                 // their ranges in the cell list
        cbase[0] = 0;
#pragma unroll
        for (int u = 0; u < NBW; ++u) {
        SM& sm = smw[u];
        const uint32_t b = b0 + u * gwarps();
        if (b >= NB) { mu[u] = 0ull; cbase[u + 1] = cbase[u]; continue; }
        // ---- stage the 2n+1 rows (LDGSTS: 16 bytes per lane = one 512-byte row per warp instruction,
        // no register round trip); a missing neighbour brick is zero-filled by the same instruction.
        const uint32_t my_row = nx_row[u];
        const uint64_t my_mask = nx_mask[u], bk = nx_bk[u];
        // (a missing brick copies nothing and zero-fills: the source address is then only a placeholder)
        if (ALL2) {
            // one combined row per dimension: lane L copies the 16-byte chunk of slots 2L, 2L + 1 from the lower
            // neighbour's row if bit j of those slots is set, from the upper neighbour's row otherwise; in the last
            // dimension (stride 1) the two slots of a chunk differ in that bit: two 8-byte copies
#pragma unroll
            for (int j = 0; j < NDIM; ++j) {
                if (G::SH(j) >= 1) {
                    const int side = (((2 * (int)lane) >> G::SH(j)) & 1) ? 0 : 1;       // 0: lower neighbour (d = 2j), 1: upper
                    const uint32_t row = __shfl_sync(0xffffffffu, my_row, 2 * j + side);
                    __pipeline_memcpy_async(&sm.R[j][2 * lane], reinterpret_cast<const void*>(qlane + (uint64_t)(row == NBR_NONE ? b : row) * 512ull), 16, row == NBR_NONE ? 16 : 0);
                } else {
                    const uint32_t rl = __shfl_sync(0xffffffffu, my_row, 2 * j), ru = __shfl_sync(0xffffffffu, my_row, 2 * j + 1);
                    __pipeline_memcpy_async(&sm.R[j][2 * lane], reinterpret_cast<const void*>(qlane + (uint64_t)(ru == NBR_NONE ? b : ru) * 512ull), 8, ru == NBR_NONE ? 8 : 0);
                    __pipeline_memcpy_async(&sm.R[j][2 * lane + 1], reinterpret_cast<const void*>(qlane + 8ull + (uint64_t)(rl == NBR_NONE ? b : rl) * 512ull), 8, rl == NBR_NONE ? 8 : 0);
                }
            }
            __pipeline_memcpy_async(&sm.R[OWN][2 * lane], reinterpret_cast<const void*>(qlane + (uint64_t)b * 512ull), 16);
            if (lane < ND) sm.adjr[lane] = my_row;
        } else {
#pragma unroll
            for (int r = 0; r < SM::ROWS; ++r) {
                const uint32_t row = __shfl_sync(0xffffffffu, my_row, r);
                __pipeline_memcpy_async(&sm.R[r][2 * lane], reinterpret_cast<const void*>(qlane + (uint64_t)(row == NBR_NONE ? b : row) * 512ull), 16, row == NBR_NONE ? 16 : 0);
            }
        }
        // ---- while the rows are in flight: activity masks, coordinate tables, face array, cell list
        const uint64_t m = ((uint64_t)__shfl_sync(0xffffffffu, (uint32_t)(my_mask >> 32), LOWN) << 32) |
                           __shfl_sync(0xffffffffu, (uint32_t)my_mask, LOWN);
        if (lane < ND) {
            const bool up = lane & 1;
            const unsigned long long a1 = ((up ? m >> my_s : m << my_s) & ~my_edge) |
                                          ((up ? my_mask << my_w : my_mask >> my_w) & my_edge);
            const unsigned long long a2 = ((up ? m >> 2 * my_s : m << 2 * my_s) & ~my_edge2) |
                                          ((up ? my_mask << my_w2 : my_mask >> my_w2) & my_edge2);
            sm.A[lane] = a1;
            sm.RZ[lane] = nolim ? m & ~a1 : m & ~a1 & a2;      // without a limiter the wave needs no second cell
        }
        for (int t = (int)lane; t < FG::NF; t += 32) {
            int tj = 0, ti = t;
#pragma unroll
            for (int j = 1; j < NDIM; ++j) if (t >= FG::XF(j)) { tj = j; ti = t - FG::XF(j); }
            const int sh = (NDIM - 1 - tj) * p.bits;
            const int32_t Bj = (int32_t)((int64_t)((bk >> sh) & ((1ull << p.bits) - 1ull)) - p.bias);
            int kk = 0;
#pragma unroll
            for (int j = 0; j < NDIM; ++j) if (tj == j) kk = G::K(j);
            const double ci = (double)(Bj * (1 << kk) + ti);
            const double hj = p.h[tj], mj = p.mu[tj];
            sm.xf[t] = DADD(mj, DMUL(ci - 0.5, hj));
            if (ti < (1 << kk)) sm.xc[t - tj] = DADD(mj, DMUL(ci, hj));
        }
#pragma unroll
        for (int j = 0; j < NDIM; ++j)
            if (2 * (int)lane < FG::FB) *reinterpret_cast<double2*>(&sm.Fb[j][2 * lane]) = make_double2(0.0, 0.0);
        const uint32_t m_lo = (uint32_t)m, m_hi = (uint32_t)(m >> 32);
        const uint32_t below = (1u << lane) - 1u;
        if ((m_lo >> lane) & 1u) wlist[cbase[u] + __popc(m_lo & below)] = (uint8_t)((u << 6) | lane);
        if ((m_hi >> lane) & 1u) wlist[cbase[u] + __popc(m_lo) + __popc(m_hi & below)] = (uint8_t)((u << 6) | (lane + 32));
        mu[u] = m;
        cbase[u + 1] = cbase[u] + __popcll(m);
        }
        __pipeline_commit();
        fetch_rows(b0 + NBW * gwarps());                    // next round: rows now, masks after the cell loop
        const int cnt = cbase[NBW];
        ncells += (unsigned)cnt;
        __pipeline_wait_prior(0);
        __syncwarp();
        // ---- cell loop: active cells, 32 at a time
        for (int r0 = 0; r0 < cnt; r0 += 32) {
            if (r0 + (int)lane >= cnt) continue;
            const unsigned e = wlist[r0 + lane];
            const int l = (int)(e & 63u);
            SM& cs = smw[NBW > 1 ? (e >> 6) : 0];           // the cell's brick
            const uint32_t b = b0 + (NBW > 1 ? (e >> 6) : 0u) * gwarps();
            const double* Rf = &cs.R[0][0];
            const double q0 = cs.R[OWN][l];
            const unsigned lbit = 1u << (l & 31);
            const unsigned* Aw = reinterpret_cast<const unsigned*>(&cs.A[0]) + (l >> 5);    // this cell's half of every mask
            const unsigned* Zw = reinterpret_cast<const unsigned*>(&cs.RZ[0]) + (l >> 5);
            double x[NDIM], al[NDIM], au[NDIM], dm[NDIM], dp[NDIM], T[NDIM];
#pragma unroll
            for (int j = 0; j < NDIM; ++j) x[j] = cs.xc[FG::XC(j) + ((l >> G::SH(j)) & G::MK(j))];
            double S = 0.0;
#pragma unroll
            for (int j = 0; j < NDIM; ++j) {
                const int s = 1 << G::SH(j), MK = G::MK(j);
                const int lj = (l >> G::SH(j)) & MK;
                const double tA = __dmul_rn(tau[j], (dyn_A<NDIM, DYN>(p, x, j)));
                al[j] = __fma_rn(tauB[j], cs.xf[FG::XF(j) + lj], tA);
                au[j] = __fma_rn(tauB[j], cs.xf[FG::XF(j) + lj + 1], tA);
                double vm, vp;
                if (ALL2) {                        // both neighbours sit at slot l ^ s: one in the own row, one in the combined row j
                    const double v_in = Rf[OWN * 64 + (l ^ s)], v_out = Rf[j * 64 + (l ^ s)];
                    vm = lj ? v_in : v_out;
                    vp = lj ? v_out : v_in;
                } else if (G::K(j) == 1) {         // two cells along j: both neighbours sit at slot l ^ s, in the own row or across the face
                    const double* nb = Rf + (l ^ s);
                    vm = nb[(lj ? OWN : 2 * j) * 64];
                    vp = nb[(lj ? 2 * j + 1 : OWN) * 64];
                } else {
                    vm = Rf[lj > 0 ? OWN * 64 + l - s : (2 * j) * 64 + l + MK * s];
                    vp = Rf[lj < MK ? OWN * 64 + l + s : (2 * j + 1) * 64 + l - MK * s];
                }
                dm[j] = q0 - vm;
                dp[j] = vp - q0;
                double t = 0.0;
                if (dpos(al[j])) t = al[j] * dm[j];
                if (dneg(au[j])) t = fma(au[j], dp[j], t);
                T[j] = 0.5 * t;
                S += T[j];
            }
            double part = q0;
            unsigned fl = 0;                                // bit d: fetch the flux of external face d in pass 2
            const double qS = q0 - S;
#pragma unroll
            for (int j = 0; j < NDIM; ++j) {
                const int s = 1 << G::SH(j), MK = G::MK(j);
                const int lj = (l >> G::SH(j)) & MK;
                const double Gj = qS + T[j];               // P*_{c,(j)}
                const double sig = (hires && !nolim) ? mc_limit_fast(dm[j], dp[j]) : 0.0;
                {   // upper face of c
                    const double a = au[j];
                    if (dpos(a)) {
                        const double wv = hires ? (nolim ? dp[j] : sig) : 0.0;
                        const double F = a * fma(0.5 - 0.5 * a, wv, Gj);
                        if (lj < MK) cs.Fb[j][FG::fb(j, l)] = F;
                        else {
                            part -= F;
                            if (Aw[2 * (2 * j + 1)] & lbit) st.phi[((size_t)b * ND + 2 * j + 1) * 32 + G::fidx(j, l)] = F;
                        }
                    } else if (dneg(a)) {
                        if (lj == MK && (Aw[2 * (2 * j + 1)] & lbit)) fl |= 1u << (2 * j + 1);
                        // upwind cell c+e^j inactive: W = 0 - P_c, W_up = P_{c+2e^j} - 0 (zero unless c+2e^j is active)
                        if (hires && (Zw[2 * (2 * j + 1)] & lbit)) {
                            double v2;                   // P_{c+2e^j}
                            if (nolim) v2 = 0.0;          // (not used without a limiter, and the cell behind need not exist then)
                            else if (ALL2) v2 = lj ? Q[(size_t)cs.adjr[2 * j + 1] * 64 + l] : Rf[j * 64 + l];   // upper brick, slot l: staged only for lj = 0
                            else v2 = Rf[lj + 2 <= MK ? OWN * 64 + l + 2 * s : (2 * j + 1) * 64 + l + (1 - MK) * s];
                            const double wv = nolim ? dp[j] : mc_limit_fast(dp[j], v2);
                            part -= a * ((-0.5 - 0.5 * a) * wv);
                        }
                    }
                }
                {   // lower face of c
                    const double a = al[j];
                    if (dneg(a)) {
                        const double wv = hires ? (nolim ? dm[j] : sig) : 0.0;
                        const double F = a * fma(-0.5 - 0.5 * a, wv, Gj);
                        if (lj > 0) cs.Fb[j][FG::fb(j, l - s)] = F;
                        else {
                            part += F;
                            if (Aw[2 * (2 * j)] & lbit) st.phi[((size_t)b * ND + 2 * j) * 32 + G::fidx(j, l)] = F;
                        }
                    } else if (dpos(a)) {
                        if (lj == 0 && (Aw[2 * (2 * j)] & lbit)) fl |= 1u << (2 * j);
                        // upwind cell c-e^j inactive: W = P_c - 0, W_up = 0 - P_{c-2e^j} (zero unless c-2e^j is active)
                        if (hires && (Zw[2 * (2 * j)] & lbit)) {
                            double v2;                   // P_{c-2e^j}
                            if (nolim) v2 = 0.0;
                            else if (ALL2) v2 = lj ? Rf[j * 64 + l] : Q[(size_t)cs.adjr[2 * j] * 64 + l];       // lower brick, slot l: staged only for lj = 1
                            else v2 = Rf[lj - 2 >= 0 ? OWN * 64 + l - 2 * s : (2 * j) * 64 + l + (MK - 1) * s];
                            const double wv = nolim ? dm[j] : mc_limit_fast(dm[j], -v2);
                            part += a * ((0.5 - 0.5 * a) * wv);
                        }
                    }
                }
            }
            cs.acc[l] = part;
            cs.fl[l] = (uint16_t)fl;
        }
        fetch_masks();                                      // next brick (its rows were fetched above)
        __syncwarp();
        // ---- apply the in-brick face fluxes to both of their cells, write the partial update
#pragma unroll
        for (int u = 0; u < NBW; ++u) {
        SM& sm = smw[u];
        const uint32_t b = b0 + u * gwarps();
        if (b >= NB) continue;
        const uint64_t m = mu[u];
#pragma unroll
        for (int hh = 0; hh < 2; ++hh) {
            const int l = (int)lane + 32 * hh;
            const bool on = (m >> l) & 1ull;
            double v = on ? sm.acc[l] : 0.0;
#pragma unroll
            for (int j = 0; j < NDIM; ++j) {
                const int s = 1 << G::SH(j), MK = G::MK(j);
                const int lj = (l >> G::SH(j)) & MK;
                if (G::K(j) == 1) {     // two cells along j: the one in-brick face, entered under its lower cell's slot
                    const double f = sm.Fb[j][FG::fb(j, l & ~s)];
                    v += lj ? f : -f;
                } else {
                    if (lj < MK) v -= sm.Fb[j][FG::fb(j, l)];
                    if (lj > 0) v += sm.Fb[j][FG::fb(j, l - s)];
                }
            }
            st.Qn[(size_t)b * 64 + l] = on ? v : 0.0;
            st.fetch[(size_t)b * 64 + l] = on ? sm.fl[l] : (uint16_t)0;
        }
        }
        __syncwarp();
    }
    if (lane == 0 && ncells) atomicAdd(&ds->Ncount, (unsigned long long)ncells);
}

// ---- a5+a6 pass 2: fetch the fluxes owned by neighbour bricks, finish the update, sum the mass --
template <int NDIM>
__device__ void phase_flux2(const Params& p, const Store& st, DevState* ds) {
    using G = Geo<NDIM>;
    constexpr int ND = 2 * NDIM;
    const uint32_t NB = min(ds->NB, p.capB);
    const unsigned lane = lane_id();
    double sum = 0.0;
    for (uint32_t b = gwarp(); b < NB; b += gwarps()) {
        uint32_t my_nb = NBR_NONE;
        if (lane < ND) my_nb = st.adj[(size_t)b * ND + lane];
        double a0 = st.Qn[(size_t)b * 64 + lane], a1 = st.Qn[(size_t)b * 64 + 32 + lane];
        const unsigned f0 = st.fetch[(size_t)b * 64 + lane], f1 = st.fetch[(size_t)b * 64 + 32 + lane];
        const unsigned any = __reduce_or_sync(0xffffffffu, f0 | f1);
        if (any) {
#pragma unroll
            for (int d = 0; d < ND; ++d) {
                if (!((any >> d) & 1u)) continue;
                const uint32_t nb = __shfl_sync(0xffffffffu, my_nb, d);
                const int j = d >> 1;
                const double* src = st.phi + ((size_t)nb * ND + (d ^ 1)) * 32;
                if ((f0 >> d) & 1u) { const double v = src[G::fidx(j, (int)lane)]; a0 += (d & 1) ? -v : v; }
                if ((f1 >> d) & 1u) { const double v = src[G::fidx(j, (int)lane + 32)]; a1 += (d & 1) ? -v : v; }
            }
            st.Qn[(size_t)b * 64 + lane] = a0;
            st.Qn[(size_t)b * 64 + 32 + lane] = a1;
        }
        sum += a0 + a1;
    }
    sum = block_sum(sum);
    if (threadIdx.x == 0) st.partial[blockIdx.x] = sum;
}

// plain sum of Q and recount of the active cells (init / import / correct / prune)
__device__ inline void phase_sum(const Params& p, const Store& st, DevState* ds, bool count) {
    const uint32_t NB = min(ds->NB, p.capB);
    const uint64_t items = (uint64_t)NB * 64;
    double sum = 0.0;
    for (uint64_t i = gtid(); i < items; i += gthreads()) sum += st.Q[i];
    sum = block_sum(sum);
    if (threadIdx.x == 0) st.partial[blockIdx.x] = sum;
    if (count) {
        double n = 0.0;
        for (uint32_t b = gtid(); b < NB; b += gthreads()) n += (double)__popcll(st.mask[b]);
        n = block_sum(n);
        if (threadIdx.x == 0 && n > 0.0) atomicAdd(&ds->N, (unsigned long long)n);
    }
}

// decide on the device whether the next enqueued step executes, and set it up (thread 0 of one block)
__device__ __forceinline__ void begin_step(DevState* ds) {
    const double t = ds->t, tt = ds->t_target;
    ds->go = (t < tt) && (ds->steps < ds->step_limit) && ds->err == 0 && ds->N > 0ull;
    ds->dt_cap = tt < 1e299 ? tt - t : 0.0;
    ds->N_before_grow = ds->N;
    ds->NB_before_grow = ds->NB;
    ds->nsrc = 0u;
}

// one block: add the partials in index order, set the scale. after_step: advance t, count, flip
// the Q/Qn parity (pass 2 left the new masses in Qn) and set up the next step.
__device__ inline void finish_sum(const Params& p, const Store& st, DevState* ds, unsigned nparts, bool after_step) {
    double v = 0.0;
    for (unsigned k = threadIdx.x; k < nparts; k += blockDim.x) v += st.partial[k];
    v = block_sum(v);
    if (threadIdx.x == 0) {
        // one thread closes the step: every field it needs is read up front (one round trip to L2 instead
        // of a chain of them), the updates are plain stores
        const double old = ds->scale, t0 = ds->t, tt = ds->t_target, cap = ds->dt_cap;
        const unsigned long long N0 = ds->N, Nc = ds->Ncount, Nbg = ds->N_before_grow, steps = ds->steps,
                                 limit = ds->step_limit, upd = ds->cell_updates, ins = ds->inserted_total,
                                 sbits = ds->smax_bits;
        const unsigned parity = ds->parity;
        const uint32_t NBc = ds->NB;
        int err = ds->err;
        ds->sumQ = v;
        if (!(v > 0.0) || !isfinite(v)) {
            if (p.normalise || !isfinite(v)) err |= E_DEGENERATE;
        }
        ds->mass = v * old;
        if (p.normalise && v > 0.0) ds->scale = 1.0 / v;
        const unsigned long long N = after_step ? Nc : N0;      // pass 1 counted the grown grid
        if (N > p.max_cells) err |= E_CAPACITY;
        if (after_step) {
            const double smax = __longlong_as_double((long long)sbits);
            const bool capped = isfinite(cap) && cap > 0.0;      // same arithmetic as step_dt()
            double dt = smax > 0.0 ? __ddiv_rn(p.cfl, smax) : (capped ? cap : 0.0);
            if (capped && cap < dt) dt = cap;
            if (!(dt > 0.0)) err |= E_DEGENERATE;
            const double t1 = t0 + dt;
            ds->N = N;
            ds->Ncount = 0ull;
            ds->dt = dt;
            ds->t = t1;
            ds->steps = steps + 1;
            ds->cell_updates = upd + N;
            ds->inserted_total = ins + (N - Nbg);
            ds->parity = parity ^ 1u;
            ds->prune_ok = 1;
            // begin_step() for the next step, from the values at hand
            ds->go = (t1 < tt) && (steps + 1 < limit) && err == 0 && N > 0ull;
            ds->dt_cap = tt < 1e299 ? tt - t1 : 0.0;
            ds->N_before_grow = N;
            ds->NB_before_grow = NBc;
            ds->nsrc = 0u;
        }
        if (err) atomicOr(&ds->err, err);
    }
}

// pass 2 + mass sum + step bookkeeping in one launch: the last block to finish (ticket) adds the
// per-block partials in index order (deterministic) and closes the step.
template <int NDIM>
__device__ void phase_flux2_finish(const Params& p, const Store& st, DevState* ds) {
    __shared__ bool s_last;
    phase_flux2<NDIM>(p, st, ds);
    if (threadIdx.x == 0) {
        __threadfence();
        s_last = atomicAdd(&ds->ticket, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (s_last) {
        __threadfence();
        finish_sum(p, st, ds, gridDim.x, true);
        if (threadIdx.x == 0) ds->ticket = 0;
    }
}

// ---- a7 prune, D3 (Alg. 3) -------------------------------------------
// mark = phase_targets<.., false>. Then: new mask = mask & keep; bricks left without a cell are
// freed; surviving bricks are stream-compacted (decoupled-lookback scan over BRICKS), removed cells
// are zeroed, the table is rebuilt and the adjacency re-linked.
__device__ inline void phase_prune_scan(const Params& p, const Store& st, DevState* ds) {
    const uint32_t NB = min(ds->NB, p.capB);
    if (NB == 0) { if (gtid() == 0) ds->NB_after_prune = 0; return; }
    scan_compact(
        NB, st.tile_state, &ds->tile_counter, &ds->NB_after_prune,
        [&](uint32_t i) { return (st.mask[i] & st.keep[i]) != 0ull; },
        [&](uint32_t i, uint32_t d) {
            st.newrow[i] = d;
            st.bkey2[d] = st.bkey[i];
            st.mask2[d] = st.mask[i] & st.keep[i];
        },
        [&](uint32_t i) { st.newrow[i] = NBR_NONE; });
}

// move the surviving bricks' rows (Q -> Qn at the new row), zero removed cells, keep the GROWN bit
// only for cells still >= p* (their targets were all kept)
__device__ inline void phase_prune_move(const Params& p, const Store& st, DevState* ds) {
    const uint32_t NB = min(ds->NB, p.capB);
    const double scale = ds->scale, thresh = p.thresh;
    const unsigned lane = lane_id();
    for (uint32_t b = gwarp(); b < NB; b += gwarps()) {
        const uint32_t d = st.newrow[b];
        if (d == NBR_NONE) continue;
        const uint64_t nm = st.mask[b] & st.keep[b];
        double q0 = st.Q[(size_t)b * 64 + lane], q1 = st.Q[(size_t)b * 64 + 32 + lane];
        if (!((nm >> lane) & 1ull)) q0 = 0.0;
        if (!((nm >> (lane + 32)) & 1ull)) q1 = 0.0;
        st.Qn[(size_t)d * 64 + lane] = q0;
        st.Qn[(size_t)d * 64 + 32 + lane] = q1;
        const uint64_t ge = (uint64_t)__ballot_sync(0xffffffffu, scale * q0 >= thresh) |
                            ((uint64_t)__ballot_sync(0xffffffffu, scale * q1 >= thresh) << 32);
        if (lane == 0) st.grown2[d] = st.grown[b] & ge & nm;
    }
}

// rows [NB_after_prune, NB) of both value buffers go back to zero (invariant: unused rows are zero)
__device__ inline void phase_zero_tail(const Params& p, const Store& st, DevState* ds) {
    const uint64_t first = (uint64_t)ds->NB_after_prune * 64, last = (uint64_t)min(ds->NB, p.capB) * 64;
    for (uint64_t i = first + gtid(); i < last; i += gthreads()) { st.Q[i] = 0.0; st.Qn[i] = 0.0; }
}

// clear the active part of the table (ds->slots was set for the new brick count)
__device__ inline void phase_clear_table(const Store& st, const DevState* ds) {
    const uint64_t slots = ds->slots;
    const ulonglong2 e = make_ulonglong2(KEY_EMPTY, KEY_EMPTY);
    for (uint64_t s = gtid(); s < slots; s += gthreads()) { st.table[s] = e; st.pend[s] = 0ull; }
}

// insert every brick key with its row (table was cleared)
__device__ inline void phase_rebuild(const Params& p, const Store& st, DevState* ds) {
    const uint32_t NB = min(ds->NB, p.capB);
    const uint64_t slots = ds->slots;
    for (uint32_t i = gtid(); i < NB; i += gthreads()) {
        const uint64_t s = ht_claim(st.table, slots, st.bkey[i]);
        if (s >= ~0ull - 1) { atomicOr(&ds->err, s == ~0ull ? E_DEGENERATE : E_TABLE_FULL); continue; }  // duplicate key
        st.table[s].y = i;
    }
}

// ---- D5 / A8 init_gaussian: one thread per candidate cell of the ellipsoid's bounding box ---------
struct GaussArgs {
    double inv[MAXN * MAXN];   // Sigma^-1 (or R^-1 for correct)
    double H[MAXN * MAXN];     // correct_linear: measurement matrix, m x n row-major
    int m;                     // correct_linear: number of measured quantities
    double v[MAXN];            // correct: measurement z (or y)
    double norm;               // P~ at the mean
    int64_t R[MAXN];           // half-extents of the bounding box in cells
    unsigned long long total;  // prod (2 R_j + 1)
};

template <int NDIM>
__device__ __forceinline__ double quad_form(const double* inv, const double d[NDIM]) {
    double q = 0.0;
#pragma unroll
    for (int i = 0; i < NDIM; ++i) {
        double r = 0.0;
#pragma unroll
        for (int j = 0; j < NDIM; ++j) r += inv[i * NDIM + j] * d[j];
        q += d[i] * r;
    }
    return q;
}

// create the brick of cell c if absent (claim + row allocation + publication). Used by init / import,
// which run the claim pass and the fill pass as separate launches.
template <int NDIM>
__device__ __forceinline__ void claim_brick(const Params& p, const Store& st, DevState* ds, const int32_t c[NDIM]) {
    constexpr int ND = 2 * NDIM;
    int32_t B[NDIM];
    cell_to_brick<NDIM>(c, B);
    const uint64_t bk = pack<NDIM>(p, B);
    bool inserted;
    const uint64_t s = ht_upsert(st.table, ds->slots, bk, inserted);
    if (s == ~0ull) { atomicOr(&ds->err, E_TABLE_FULL); return; }
    if (!inserted) return;
    const uint32_t nr = atomicAdd(&ds->NB, 1u);
    if (nr >= p.capB) { atomicOr(&ds->err, E_CAPACITY); return; }
    st.bkey[nr] = bk; st.grown[nr] = 0ull; st.mask[nr] = 0ull;
#pragma unroll
    for (int d = 0; d < ND; ++d) st.adj[(size_t)nr * ND + d] = NBR_NONE;
    st.table[s].y = nr;
}
// second pass: activate cell c with stored mass q (its brick exists)
template <int NDIM>
__device__ __forceinline__ void fill_cell(const Params& p, const Store& st, DevState* ds, const int32_t c[NDIM], double q) {
    int32_t B[NDIM];
    const int l = cell_to_brick<NDIM>(c, B);
    const uint32_t row = ht_find(st.table, ds->slots, pack<NDIM>(p, B));
    if (row == NBR_NONE || row >= p.capB) return;     // capacity error already recorded by the claim pass
    const unsigned long long bit = 1ull << l;
    if (atomicOr((unsigned long long*)&st.mask[row], bit) & bit) { atomicOr(&ds->err, E_DEGENERATE); return; }  // duplicate key
    st.Q[(size_t)row * 64 + l] = q;
}

template <int NDIM, bool FILL>
__device__ void phase_init_gaussian(const Params& p, const Store& st, DevState* ds, const GaussArgs& g) {
    const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
    for (unsigned long long r = gtid(); r < g.total; r += stride) {
        int32_t c[NDIM];
        unsigned long long rem = r;
#pragma unroll
        for (int j = NDIM - 1; j >= 0; --j) {
            const unsigned long long wd = 2ull * g.R[j] + 1ull;
            c[j] = (int32_t)((long long)(rem % wd) - g.R[j]);
            rem /= wd;
        }
        double d[NDIM];
#pragma unroll
        for (int j = 0; j < NDIM; ++j) d[j] = (double)c[j] * p.h[j];
        const double val = exp(-0.5 * quad_form<NDIM>(g.inv, d)) * g.norm;
        if (!(val >= p.thresh)) continue;
        bool ok = true;
#pragma unroll
        for (int j = 0; j < NDIM; ++j) ok = ok && c[j] >= -p.bias && c[j] <= p.bias - 1;
        if (!ok) { atomicOr(&ds->err, E_KEY_RANGE); continue; }
        if (FILL) fill_cell<NDIM>(p, st, ds, c, val);
        else claim_brick<NDIM>(p, st, ds, c);
    }
}

template <int NDIM, bool FILL>
__device__ void phase_import(const Params& p, const Store& st, DevState* ds, const int32_t* keys,
                             const double* vals, uint64_t count) {
    for (uint64_t i = gtid(); i < count; i += gthreads()) {
        int32_t c[NDIM];
        bool ok = true;
#pragma unroll
        for (int j = 0; j < NDIM; ++j) {
            c[j] = keys[(size_t)i * NDIM + j];
            ok = ok && c[j] >= -p.bias && c[j] <= p.bias - 1;
        }
        if (!ok) { atomicOr(&ds->err, E_KEY_RANGE); continue; }
        if (FILL) fill_cell<NDIM>(p, st, ds, c, vals[i]);
        else claim_brick<NDIM>(p, st, ds, c);
    }
}

// ---- a8 correct, D4 / Eq. (4): Q_c *= exp(-1/2 (z - x_c)^T R^-1 (z - x_c)) ------------
template <int NDIM>
__device__ void phase_correct(const Params& p, const Store& st, DevState* ds, const GaussArgs& g) {
    const uint32_t NB = min(ds->NB, p.capB);
    const uint64_t items = (uint64_t)NB * 64;
    for (uint64_t i = gtid(); i < items; i += gthreads()) {
        const uint32_t b = (uint32_t)(i >> 6);
        const int l = (int)(i & 63);
        if (!((st.mask[b] >> l) & 1ull)) continue;
        int32_t B[NDIM], c[NDIM];
        unpack<NDIM>(p, st.bkey[b], B);
        cell_coords<NDIM>(B, l, c);
        double d[NDIM];
#pragma unroll
        for (int j = 0; j < NDIM; ++j) d[j] = g.v[j] - (p.mu[j] + (double)c[j] * p.h[j]);
        st.Q[i] *= exp(-0.5 * quad_form<NDIM>(g.inv, d));
    }
}

// f2, Eq. (4) with y = H x + v (the paper's scenario measures x3 only):
// Q_c *= exp(-1/2 (y - H x_c)^T R^-1 (y - H x_c))
template <int NDIM>
__device__ void phase_correct_linear(const Params& p, const Store& st, DevState* ds, const GaussArgs& g) {
    const uint32_t NB = min(ds->NB, p.capB);
    const uint64_t items = (uint64_t)NB * 64;
    const int m = g.m;
    for (uint64_t i = gtid(); i < items; i += gthreads()) {
        const uint32_t b = (uint32_t)(i >> 6);
        const int l = (int)(i & 63);
        if (!((st.mask[b] >> l) & 1ull)) continue;
        int32_t B[NDIM], c[NDIM];
        unpack<NDIM>(p, st.bkey[b], B);
        cell_coords<NDIM>(B, l, c);
        double x[NDIM], d[MAXN];
#pragma unroll
        for (int j = 0; j < NDIM; ++j) x[j] = p.mu[j] + (double)c[j] * p.h[j];
#pragma unroll
        for (int r = 0; r < MAXN; ++r) {
            double hx = 0.0;
#pragma unroll
            for (int j = 0; j < NDIM; ++j) hx += g.H[r * NDIM + j] * x[j];
            d[r] = r < m ? g.v[r] - hx : 0.0;
        }
        double q = 0.0;
#pragma unroll
        for (int r = 0; r < MAXN; ++r) {
            double t = 0.0;
#pragma unroll
            for (int k = 0; k < MAXN; ++k) t += (r < m && k < m) ? g.inv[r * m + k] * d[k] : 0.0;
            q += d[r] * t;
        }
        st.Q[i] *= exp(-0.5 * q);
    }
}

// f2, a non-linear measurement: the range to a point s (g.v), y = ||x - s|| + v, v ~ N(0, sigma^2):
// Q_c *= exp(-1/2 ((y - ||x_c - s||) / sigma)^2)            (Eq. 4; g.norm = y, g.inv[0] = 1 / sigma)
template <int NDIM>
__device__ void phase_correct_range(const Params& p, const Store& st, DevState* ds, const GaussArgs& g) {
    const uint32_t NB = min(ds->NB, p.capB);
    const uint64_t items = (uint64_t)NB * 64;
    for (uint64_t i = gtid(); i < items; i += gthreads()) {
        const uint32_t b = (uint32_t)(i >> 6);
        const int l = (int)(i & 63);
        if (!((st.mask[b] >> l) & 1ull)) continue;
        int32_t B[NDIM], c[NDIM];
        unpack<NDIM>(p, st.bkey[b], B);
        cell_coords<NDIM>(B, l, c);
        double r2 = 0.0;
#pragma unroll
        for (int j = 0; j < NDIM; ++j) {
            const double d = (p.mu[j] + (double)c[j] * p.h[j]) - g.v[j];
            r2 += d * d;
        }
        const double e = (g.norm - sqrt(r2)) * g.inv[0];
        st.Q[i] *= exp(-0.5 * e * e);
    }
}

// f1, distribution metrics between two contexts on the same grid (same n, dx, origin):
//   BC = sum_c sqrt(Pa_c Pb_c)  (Eq. 9),  E = sum_c |Pa_c - Pb_c|  (masses).
// One warp per brick of A looks the brick up in B's table (hash join over BRICK keys); per-block
// partials of (BC, sum |Pa - Pb| over A's cells, sum |Pa| over A's cells that B does not have) go to
// out[3][gridDim.x]. The host runs it both ways: E = (second sum of A->B) + (third sum of B->A).
template <int NDIM>
__device__ void phase_compare(const Params& p, const Store& a, const DevState* da, const Store& b, const DevState* db,
                              double* out) {
    const uint32_t NBa = min(da->NB, p.capB);
    const double sa = da->scale, sb = db->scale;
    const uint64_t slots_b = db->slots;
    const unsigned lane = lane_id();
    double bc = 0.0, l1 = 0.0, mb = 0.0;
    for (uint32_t r = gwarp(); r < NBa; r += gwarps()) {
        const uint64_t ma = a.mask[r];
        if (!ma) continue;
        const uint32_t rb = ht_find(b.table, slots_b, a.bkey[r]);
        const uint64_t mbk = rb != NBR_NONE ? b.mask[rb] : 0ull;
#pragma unroll
        for (int hh = 0; hh < 2; ++hh) {
            const int l = (int)lane + 32 * hh;
            if (!((ma >> l) & 1ull)) continue;
            const double pa = sa * a.Q[(size_t)r * 64 + l];
            const double pb = ((mbk >> l) & 1ull) ? sb * b.Q[(size_t)rb * 64 + l] : 0.0;
            if (pa > 0.0 && pb > 0.0) bc += sqrt(pa * pb);
            l1 += fabs(pa - pb);
            if (!((mbk >> l) & 1ull)) mb += fabs(pa);
        }
    }
    bc = block_sum(bc);
    l1 = block_sum(l1);
    mb = block_sum(mb);
    if (threadIdx.x == 0) { out[blockIdx.x] = bc; out[gridDim.x + blockIdx.x] = l1; out[2 * gridDim.x + blockIdx.x] = mb; }
}

// f3, marginal PDF: the masses are hash-accumulated over the kept coordinates.
// Scratch table: skey[S] (packed kept coordinates, KEY_EMPTY = free) and sval[S] (mass), linear probing
// with the same mixer as the brick table; atomicAdd(double) accumulates, so the order of the additions
// is not fixed (rounding-level differences between runs, as the paper notes for CUDA).
struct MargArgs {
    int m;                 // kept dimensions
    int dims[MAXN];        // their indices, in output order
    int mbits;             // bits per kept coordinate in the scratch key
    unsigned long long S;  // scratch slots
};
__device__ __forceinline__ void phase_marg_clear(unsigned long long* skey, double* sval, unsigned long long S) {
    for (unsigned long long i = gtid(); i < S; i += gthreads()) { skey[i] = KEY_EMPTY; sval[i] = 0.0; }
}
template <int NDIM>
__device__ void phase_marg_accumulate(const Params& p, const Store& st, DevState* ds, const MargArgs& g,
                                      unsigned long long* skey, double* sval) {
    const uint32_t NB = min(ds->NB, p.capB);
    const uint64_t items = (uint64_t)NB * 64;
    const double scale = ds->scale;
    const long long mbias = 1ll << (g.mbits - 1);
    for (uint64_t i = gtid(); i < items; i += gthreads()) {
        const uint32_t b = (uint32_t)(i >> 6);
        const int l = (int)(i & 63);
        if (!((st.mask[b] >> l) & 1ull)) continue;
        int32_t B[NDIM], c[NDIM];
        unpack<NDIM>(p, st.bkey[b], B);
        cell_coords<NDIM>(B, l, c);
        unsigned long long key = 0ull;
        for (int r = 0; r < g.m; ++r) {
            int32_t cv = 0;
#pragma unroll
            for (int j = 0; j < NDIM; ++j) if (g.dims[r] == j) cv = c[j];
            key = (key << g.mbits) | (unsigned long long)((long long)cv + mbias);
        }
        unsigned long long s = home_slot(key, g.S);
        for (;;) {
            unsigned long long cur = *reinterpret_cast<volatile unsigned long long*>(&skey[s]);
            if (cur == KEY_EMPTY) cur = atomicCAS(&skey[s], KEY_EMPTY, key);
            if (cur == KEY_EMPTY || cur == key) break;
            if (++s == g.S) s = 0;
        }
        atomicAdd(&sval[s], scale * st.Q[i]);
    }
}
__device__ __forceinline__ void phase_marg_emit(DevState* ds, const MargArgs& g, const unsigned long long* skey,
                                                const double* sval, int32_t* keys, double* out, unsigned cap) {
    const long long mbias = 1ll << (g.mbits - 1);
    const unsigned long long fm = (1ull << g.mbits) - 1ull;
    for (unsigned long long i = gtid(); i < g.S; i += gthreads()) {
        const unsigned long long key = skey[i];
        if (key == KEY_EMPTY) continue;
        const unsigned o = atomicAdd(&ds->export_count, 1u);
        if (o >= cap) continue;
        for (int r = 0; r < g.m; ++r)
            keys[(size_t)o * g.m + r] = (int32_t)((long long)((key >> ((g.m - 1 - r) * g.mbits)) & fm) - mbias);
        out[o] = sval[i];
    }
}

// f1, spatial convergence: conservative remap of the PDF onto a grid of another origin / spacing
// (reading A19: the PDF is piecewise constant over its cells; cell d of the other grid receives P_c times the
// overlap volume fraction, a product of 1-D overlap fractions). The target grid is at least as coarse in every
// dimension, so a cell overlaps at most two target cells per dimension. Same scratch table as the marginals.
// The integer decisions (which target cells, sliver cut-off) follow the operation order DESIGN.md A19 fixes.
struct ResampleArgs {
    double o2[MAXN], h2[MAXN];
    int mbits;
    unsigned long long S;
};
template <int NDIM>
__device__ void phase_resample_accumulate(const Params& p, const Store& st, DevState* ds, const ResampleArgs& g,
                                          unsigned long long* skey, double* sval) {
    const uint32_t NB = min(ds->NB, p.capB);
    const uint64_t items = (uint64_t)NB * 64;
    const double scale = ds->scale;
    const long long mbias = 1ll << (g.mbits - 1);
    for (uint64_t i = gtid(); i < items; i += gthreads()) {
        const uint32_t b = (uint32_t)(i >> 6);
        const int l = (int)(i & 63);
        if (!((st.mask[b] >> l) & 1ull)) continue;
        int32_t B[NDIM], c[NDIM];
        unpack<NDIM>(p, st.bkey[b], B);
        cell_coords<NDIM>(B, l, c);
        const double pc = scale * st.Q[i];
        long long d0[NDIM];
        double w[NDIM][2];
        int cnt[NDIM];
#pragma unroll
        for (int j = 0; j < NDIM; ++j) {
            const double h = p.h[j], o2 = g.o2[j], h2 = g.h2[j];
            const double lo = DADD(p.mu[j], DMUL((double)c[j] - 0.5, h)), hi = DADD(p.mu[j], DMUL((double)c[j] + 0.5, h));
            const long long dl = (long long)floor(DADD(__ddiv_rn(DSUB(lo, o2), h2), 0.5));
            const long long dh = (long long)floor(DADD(__ddiv_rn(DSUB(hi, o2), h2), 0.5));
            if (dh > dl + 1) atomicOr(&ds->err, E_DEGENERATE);      // target grid finer than the source (rejected by the host)
            int n_ = 0;
            long long first = dl;
            for (int k = 0; k < 2; ++k) {
                const long long d = dl + k;
                if (d > dh) break;
                const double a = fmax(lo, DADD(o2, DMUL((double)d - 0.5, h2))), e = fmin(hi, DADD(o2, DMUL((double)d + 0.5, h2)));
                if (DSUB(e, a) > DMUL(1e-12, h)) {
                    if (n_ == 0) first = d;
                    w[j][n_++] = __ddiv_rn(DSUB(e, a), h);
                }
            }
            // target coordinates must fit the key fields of the scratch table (the width of the grid's own fields)
            if (first < -mbias || first + 1 > mbias - 1) { atomicOr(&ds->err, E_KEY_RANGE); n_ = 0; }
            d0[j] = first; cnt[j] = n_;                              // the (at most two) target cells are consecutive
            if (n_ < 2) w[j][1] = 0.0;
            if (n_ < 1) w[j][0] = 0.0;
        }
        for (int combo = 0; combo < (1 << NDIM); ++combo) {
            double wt = 1.0;
            unsigned long long key = 0ull;
            bool ok = true;
#pragma unroll
            for (int j = 0; j < NDIM; ++j) {
                const int k = (combo >> j) & 1;
                ok = ok && k < cnt[j];
                wt = DMUL(wt, k ? w[j][1] : w[j][0]);
                key = (key << g.mbits) | (unsigned long long)(d0[j] + k + mbias);
            }
            if (!ok) continue;
            unsigned long long s = home_slot(key, g.S);
            for (unsigned long long tries = 0;; ++tries) {
                if (tries == g.S) { atomicOr(&ds->err, E_TABLE_FULL); break; }
                unsigned long long cur = *reinterpret_cast<volatile unsigned long long*>(&skey[s]);
                if (cur == KEY_EMPTY) cur = atomicCAS(&skey[s], KEY_EMPTY, key);
                if (cur == KEY_EMPTY || cur == key) { atomicAdd(&sval[s], DMUL(pc, wt)); break; }
                if (++s == g.S) s = 0;
            }
        }
    }
}

// export: a warp reserves popc(mask) output rows per brick (order of bricks is unspecified)
template <int NDIM>
__device__ void phase_export(const Params& p, const Store& st, DevState* ds, int32_t* keys, double* out) {
    const uint32_t NB = min(ds->NB, p.capB);
    const double scale = ds->scale;
    const unsigned lane = lane_id();
    for (uint32_t b = gwarp(); b < NB; b += gwarps()) {
        const uint64_t m = st.mask[b];
        const int cnt = __popcll(m);
        if (cnt == 0) continue;
        unsigned base = 0;
        if (lane == 0) base = atomicAdd(&ds->export_count, (unsigned)cnt);
        base = __shfl_sync(0xffffffffu, base, 0);
        int32_t B[NDIM];
        unpack<NDIM>(p, st.bkey[b], B);
#pragma unroll
        for (int hh = 0; hh < 2; ++hh) {
            const int l = (int)lane + 32 * hh;
            if (!((m >> l) & 1ull)) continue;
            const size_t o = base + (unsigned)__popcll(m & ((1ull << l) - 1ull));
            if (keys) {
                int32_t c[NDIM];
                cell_coords<NDIM>(B, l, c);
#pragma unroll
                for (int j = 0; j < NDIM; ++j) keys[o * NDIM + j] = c[j];
            }
            if (out) out[o] = scale * st.Q[(size_t)b * 64 + l];
        }
    }
}

}  // namespace gbees
