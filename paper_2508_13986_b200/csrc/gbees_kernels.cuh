// Kernels of the GBEES prediction step. Every phase is a grid-stride __device__ function so the
// same code runs as a stream of small launches (gbees_step) or inside the persistent cooperative
// loop (gbees_run). Semantics: DESIGN.md D1-D5; layout: DESIGN.md "Data layout".
#pragma once
#include "gbees_common.cuh"

namespace gbees {

constexpr int TPB = 256;

__device__ __forceinline__ unsigned gtid() { return blockIdx.x * blockDim.x + threadIdx.x; }
__device__ __forceinline__ unsigned gthreads() { return gridDim.x * blockDim.x; }

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ double warp_max(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
// block-wide sum, result valid in thread 0. Fixed order => deterministic for a fixed launch shape.
__device__ __forceinline__ double block_sum(double v) {
    __shared__ double sh[32];
    __syncthreads();
    v = warp_sum(v);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
    __syncthreads();
    double r = 0.0;
    if (threadIdx.x < 32) {
        r = threadIdx.x < (blockDim.x >> 5) ? sh[threadIdx.x] : 0.0;
        r = warp_sum(r);
    }
    return r;
}
__device__ __forceinline__ double block_max(double v) {
    __shared__ double shm[32];
    __syncthreads();
    v = warp_max(v);
    if ((threadIdx.x & 31) == 0) shm[threadIdx.x >> 5] = v;
    __syncthreads();
    double r = 0.0;
    if (threadIdx.x < 32) {
        r = threadIdx.x < (blockDim.x >> 5) ? shm[threadIdx.x] : 0.0;
        r = warp_max(r);
    }
    return r;
}

// ---- Targets(c), D1.1 / A10 / A11: downwind face + pairwise-edge neighbours -------------------
// fn(key, in_range). Range: a coordinate must stay inside the packable field.
template <int NDIM, typename F>
__device__ __forceinline__ void for_each_target(const Params& p, uint64_t key, const int32_t c[NDIM],
                                                const double ul[NDIM], const double uu[NDIM], F&& fn) {
    const int32_t lo = (int32_t)(-p.bias), hi = (int32_t)(p.bias - 1);
    // per dim: bit0 = outflow through lower face (u<0), bit1 = outflow through upper face (u>0)
    int o[NDIM];
#pragma unroll
    for (int j = 0; j < NDIM; ++j) o[j] = (ul[j] < 0.0 ? 1 : 0) | (uu[j] > 0.0 ? 2 : 0);
#pragma unroll
    for (int j = 0; j < NDIM; ++j) {
        const uint64_t uj = 1ull << ((NDIM - 1 - j) * p.bits);
#pragma unroll
        for (int sj = 0; sj < 2; ++sj) {
            if (!(o[j] & (1 << sj))) continue;
            const bool okj = sj ? (c[j] < hi) : (c[j] > lo);
            const uint64_t kj = sj ? key + uj : key - uj;
            fn(kj, okj);
#pragma unroll
            for (int l = j + 1; l < NDIM; ++l) {
                const uint64_t ulk = 1ull << ((NDIM - 1 - l) * p.bits);
#pragma unroll
                for (int sl = 0; sl < 2; ++sl) {
                    if (!(o[l] & (1 << sl))) continue;
                    const bool okl = sl ? (c[l] < hi) : (c[l] > lo);
                    fn(sl ? kj + ulk : kj - ulk, okj && okl);
                }
            }
        }
    }
}

// ---- a1 grow (Alg. 2 without staging: atomicCAS claims the slot) ------
// Targets are numbered t in [0, 2n + 4 C(n,2)): t < 2n is the face target (dim t>>1, side t&1);
// the rest are edge targets (pair (j<l), side_j, side_l).
template <int NDIM>
struct TargetTable {
    static constexpr int NT = 2 * NDIM + 2 * NDIM * (NDIM - 1);
};
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

// Block-cooperative: cells that newly need growing are compacted into shared memory, then the
// (cell, target) pairs are spread over all threads, so one front cell's ~n + C(n,2) dependent
// hashtable claims do not serialise on a single lane.
template <int NDIM, int DYN>
__device__ void phase_grow(const Params& p, const Pool& pool, DevState* st) {
    constexpr int NT = TargetTable<NDIM>::NT;
    __shared__ uint64_t s_key[TPB];
    __shared__ uint32_t s_flag[TPB];   // bits [0,2n): outflow (2j: lower, 2j+1: upper); [16,16+2n): at range border
    __shared__ unsigned s_cnt;
    const uint32_t N0 = st->N_before_grow;
    const double scale = st->scale;
    const uint64_t slots = st->slots;
    const int32_t lo = (int32_t)(-p.bias), hi = (int32_t)(p.bias - 1);
    for (uint32_t base = blockIdx.x * blockDim.x; base < N0; base += gthreads()) {
        if (threadIdx.x == 0) s_cnt = 0;
        __syncthreads();
        const uint32_t i = base + threadIdx.x;
        if (i < N0) {
            const uint64_t kf = pool.key[i];
            if (!(kf & KEY_GROWN) && scale * pool.Q[i] >= p.thresh) {   // autonomous f: grow once
                int32_t c[NDIM];
                unpack<NDIM>(p, kf, c);
                double ul[NDIM], uu[NDIM];
                face_velocities<NDIM, DYN>(p, c, ul, uu);
                uint32_t f = 0;
#pragma unroll
                for (int j = 0; j < NDIM; ++j) {
                    f |= (ul[j] < 0.0 ? 1u : 0u) << (2 * j);
                    f |= (uu[j] > 0.0 ? 1u : 0u) << (2 * j + 1);
                    f |= (c[j] <= lo ? 1u : 0u) << (16 + 2 * j);
                    f |= (c[j] >= hi ? 1u : 0u) << (16 + 2 * j + 1);
                }
                const unsigned k = atomicAdd(&s_cnt, 1u);
                s_key[k] = kf;
                s_flag[k] = f;
                pool.key[i] = kf | KEY_GROWN;
            }
        }
        __syncthreads();
        const unsigned total = s_cnt * NT;
        for (unsigned w = threadIdx.x; w < total; w += blockDim.x) {
            const unsigned cell = w / NT;
            const int t = (int)(w - cell * NT);
            int j, sj, l, sl;
            decode_target<NDIM>(t, j, sj, l, sl);
            const uint32_t f = s_flag[cell];
            if (!((f >> (2 * j + sj)) & 1u)) continue;
            if (l >= 0 && !((f >> (2 * l + sl)) & 1u)) continue;
            bool bad = (f >> (16 + 2 * j + sj)) & 1u;
            if (l >= 0) bad = bad || ((f >> (16 + 2 * l + sl)) & 1u);
            if (bad) { atomicOr(&st->err, E_KEY_RANGE); continue; }
            uint64_t tk = s_key[cell];
            const uint64_t uj = 1ull << ((NDIM - 1 - j) * p.bits);
            tk = sj ? tk + uj : tk - uj;
            if (l >= 0) {
                const uint64_t ulk = 1ull << ((NDIM - 1 - l) * p.bits);
                tk = sl ? tk + ulk : tk - ulk;
            }
            const uint64_t s = ht_claim(pool.table, slots, tk);
            if (s == ~0ull) continue;                 // already there
            if (s == ~0ull - 1) { atomicOr(&st->err, E_TABLE_FULL); continue; }
            const uint32_t idx = atomicAdd(&st->N, 1u);
            if (idx >= p.cap) { atomicOr(&st->err, E_CAPACITY); pool.table[s].y = NBR_NONE; continue; }
            pool.table[s].y = idx;
            pool.key[idx] = tk;
            pool.Q[idx] = 0.0;
#pragma unroll
            for (int d = 0; d < 2 * NDIM; ++d) pool.nbr[(size_t)d * p.cap + idx] = NBR_NONE;
        }
        __syncthreads();
    }
}

// ---- adjacency + CFL term of the linked cells -----------------------------------
// ALL = true: rebuild for every cell (after init / import / prune); false: only cells created by
// this step's grow, which also patch the slots of their neighbours. atomicMin makes a direct
// index (< NBR_TAG) win over a tagged two-hop index, which wins over NBR_NONE.
template <int NDIM, int DYN, bool ALL>
__device__ void phase_link(const Params& p, const Pool& pool, DevState* st) {
    const uint32_t first = ALL ? 0u : st->N_before_grow;
    const uint32_t N = min(st->N, p.cap);
    const uint32_t cnt = N - first;
    const uint64_t slots = st->slots;
    const int32_t lo = (int32_t)(-p.bias), hi = (int32_t)(p.bias - 1);
    // one work item per (direction, cell), direction-major: coalesced adjacency writes and the
    // 2n dependent lookups of a cell run on 2n different threads
    const uint64_t items = (uint64_t)cnt * (2 * NDIM);
    for (uint64_t w = gtid(); w < items; w += gthreads()) {
        const int d = (int)(w / cnt);
        const uint32_t i = first + (uint32_t)(w - (uint64_t)d * cnt);
        const int j = d >> 1, s = d & 1, od = d ^ 1;
        const uint64_t key = pool.key[i] & ~KEY_GROWN;
        const uint64_t uj = 1ull << ((NDIM - 1 - j) * p.bits);
        const int32_t cj = (int32_t)((int64_t)((key >> ((NDIM - 1 - j) * p.bits)) & ((1ull << p.bits) - 1ull)) - p.bias);
        uint32_t val = NBR_NONE;
        if (s ? (cj < hi) : (cj > lo)) {
            const uint32_t nb = ht_find(pool.table, slots, s ? key + uj : key - uj);
            if (nb != NBR_NONE) {
                val = nb;
                if (!ALL) atomicMin(&pool.nbr[(size_t)od * p.cap + nb], i);
            } else if (s ? (cj < hi - 1) : (cj > lo + 1)) {
                const uint32_t nb2 = ht_find(pool.table, slots, s ? key + 2 * uj : key - 2 * uj);
                if (nb2 != NBR_NONE) {
                    val = NBR_TAG | nb2;
                    if (!ALL) atomicMin(&pool.nbr[(size_t)od * p.cap + nb2], NBR_TAG | i);
                }
            }
        }
        uint32_t* mine = &pool.nbr[(size_t)d * p.cap + i];
        if (ALL) *mine = val;
        else if (val != NBR_NONE) atomicMin(mine, val);
    }
    // CFL term of the linked cells (Eq. 8): running maximum
    double smax = 0.0;
    for (uint32_t i = first + gtid(); i < N; i += gthreads()) {
        int32_t c[NDIM];
        unpack<NDIM>(p, pool.key[i] & ~KEY_GROWN, c);
        double ul[NDIM], uu[NDIM];
        face_velocities<NDIM, DYN>(p, c, ul, uu);
        smax = fmax(smax, cfl_term<NDIM>(p, ul));
    }
    smax = block_max(smax);
    if (threadIdx.x == 0 && smax > 0.0) atomicMax(&st->smax_bits, (unsigned long long)__double_as_longlong(smax));
}

// dt of Eq. (8) with the caller's cap (every thread computes the same value)
__device__ __forceinline__ double step_dt(const Params& p, const DevState* st) {
    const double smax = __longlong_as_double((long long)st->smax_bits);
    const double cap = st->dt_cap;
    const bool capped = isfinite(cap) && cap > 0.0;
    double dt = smax > 0.0 ? __ddiv_rn(p.cfl, smax) : (capped ? cap : 0.0);
    if (capped && cap < dt) dt = cap;
    return dt;
}

// ---- a2+a4 pass A: every active cell computes the fluxes of the faces it is UPWIND of -----------
// Gather form D2 (= Eq. 7 + Alg. 1 + high-resolution term):
//   T_l   = u+_{c,l}(P_c - P_{c-e^l}) + u-_{c+e^l,l}(P_{c+e^l} - P_c)
//   G_j   = P*_{c,(j)} = P_c - sum_{l != j} 1/2 tau_l T_l
//   sig_j = mc(P_c - P_{c-e^j}, P_{c+e^j} - P_c)     (limited wave when c is the upwind cell)
//   upper face, u = u_{c+e^j,j} > 0:  F = u (G_j + 1/2 (1 - tau_j u) sig_j)
//   lower face, u = u_{c,j}     < 0:  F = u (G_j - 1/2 (1 + tau_j u) sig_j)
// A face whose upwind cell is NOT active carries only the high-resolution term; the active
// downwind cell computes it (needs the two-hop value through the tagged adjacency slot).
// acc_c = P_c - sum_j tau_j (F_up - F_lo) over the faces computed here; tau_j F is stored for the
// neighbour that shares the face; mask tells pass B which faces to fetch from neighbours.
// Thread mapping: one WARP per (tile of 32 cells, dimension j). The NDIM warps of a tile exchange
// T_l and their partial updates through shared memory, so a thread holds the state of one cell in
// one dimension only (few registers, 6x the threads in flight, coalesced adjacency loads).
template <int NDIM> struct PassACfg {
    static constexpr int GROUPS = NDIM == 1 ? 8 : NDIM == 2 ? 4 : NDIM == 3 ? 2 : NDIM == 4 ? 2 : 1;
    static constexpr int BLK = 32 * NDIM * GROUPS;   // 256, 256, 192, 256, 160, 192
};

struct PassALocal {
    double q0, vm, vp, ul, uu, dm, dp, T, tau;
    uint32_t nbm, nbp, i;
    bool valid;
};

template <int NDIM, int DYN, int J>
__device__ __forceinline__ void passA_stage1(const Params& p, const Pool& pool, PassALocal& L) {
    const size_t cap = p.cap;
    const uint64_t key = pool.key[L.i] & ~KEY_GROWN;
    L.q0 = pool.Q[L.i];
    L.nbm = pool.nbr[(size_t)(2 * J) * cap + L.i];
    L.nbp = pool.nbr[(size_t)(2 * J + 1) * cap + L.i];
    L.vm = L.nbm != NBR_NONE ? pool.Q[L.nbm & ~NBR_TAG] : 0.0;   // tagged slot: the two-hop value
    L.vp = L.nbp != NBR_NONE ? pool.Q[L.nbp & ~NBR_TAG] : 0.0;
    int32_t c[NDIM];
    unpack<NDIM>(p, key, c);
    double x[NDIM];
#pragma unroll
    for (int m = 0; m < NDIM; ++m) x[m] = DADD(p.mu[m], DMUL((double)c[m], p.h[m]));
    L.ul = dyn_f<NDIM, DYN>(p, x, J, DADD(p.mu[J], DMUL((double)c[J] - 0.5, p.h[J])));
    L.uu = dyn_f<NDIM, DYN>(p, x, J, DADD(p.mu[J], DMUL((double)c[J] + 0.5, p.h[J])));
    L.dm = L.q0 - (L.nbm < NBR_TAG ? L.vm : 0.0);
    L.dp = (L.nbp < NBR_TAG ? L.vp : 0.0) - L.q0;
    double t = 0.0;
    if (L.ul > 0.0) t = L.ul * L.dm;
    if (L.uu < 0.0) t = fma(L.uu, L.dp, t);
    L.T = (0.5 * L.tau) * t;
}

// faces of dimension J owned by this cell; returns the partial update (-F_up + F_lo) and mask bits
template <int J>
__device__ __forceinline__ double passA_stage2(const Params& p, const Pool& pool, const PassALocal& L, double S,
                                               unsigned& mask) {
    const size_t cap = p.cap;
    const bool hires = p.hi_res != 0, nolim = p.limiter != 0;
    const double G = (L.q0 - S) + L.T;     // P*_{c,(J)} = q0 - sum_{l != J} T_l
    const double sig = (hires && !nolim) ? mc_limit_fast(L.dm, L.dp) : 0.0;
    const double tau = L.tau;
    double part = 0.0;
    {   // upper face of c
        const double u = L.uu;
        if (u > 0.0) {
            const double a = tau * u;
            const double w = hires ? (nolim ? L.dp : sig) : 0.0;
            const double F = a * fma(0.5 * (1.0 - a), w, G);
            part -= F;
            if (L.nbp < NBR_TAG) pool.phi[(size_t)(2 * J + 1) * cap + L.i] = F;
        } else if (u < 0.0) {
            if (L.nbp < NBR_TAG) {
                mask |= 1u << (8 + J);
            } else if (hires) {   // upwind cell c+e^J inactive: W = 0 - P_c, W_up = P_{c+2e^J} - 0
                const double w = nolim ? -L.q0 : mc_limit(-L.q0, L.vp);
                const double a = tau * u;
                part -= (-0.5 * a) * (1.0 + a) * w;
            }
        }
    }
    {   // lower face of c
        const double u = L.ul;
        if (u < 0.0) {
            const double a = tau * u;
            const double w = hires ? (nolim ? L.dm : sig) : 0.0;
            const double F = a * fma(-0.5 * (1.0 + a), w, G);
            part += F;
            if (L.nbm < NBR_TAG) pool.phi[(size_t)(2 * J) * cap + L.i] = F;
        } else if (u > 0.0) {
            if (L.nbm < NBR_TAG) {
                mask |= 1u << J;
            } else if (hires) {   // upwind cell c-e^J inactive: W = P_c - 0, W_up = 0 - P_{c-2e^J}
                const double w = nolim ? L.q0 : mc_limit(L.q0, -L.vm);
                const double a = tau * u;
                part += (0.5 * a) * (1.0 - a) * w;
            }
        }
    }
    return part;
}

template <int NDIM, int DYN>
__device__ void phase_passA(const Params& p, const Pool& pool, DevState* st) {
    constexpr int GROUPS = PassACfg<NDIM>::GROUPS;
    __shared__ double sT[GROUPS][NDIM][32];
    __shared__ double sPart[GROUPS][NDIM][32];
    __shared__ unsigned sMask[GROUPS][NDIM][32];
    const uint32_t N = min(st->N, p.cap);
    const double dt = step_dt(p, st);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int grp = warp / NDIM, j = warp - grp * NDIM;
    const uint32_t tiles = (N + 31) >> 5;
    PassALocal L;
    L.tau = dt / p.h[j];
    for (uint32_t tb = blockIdx.x * GROUPS; tb < tiles; tb += gridDim.x * GROUPS) {   // block-uniform
        const uint32_t tile = tb + grp;
        L.i = tile * 32 + lane;
        L.valid = grp < GROUPS && L.i < N;
        L.T = 0.0;
        if (L.valid) {
            switch (j) {
                case 0: passA_stage1<NDIM, DYN, 0>(p, pool, L); break;
                case 1: if constexpr (NDIM > 1) passA_stage1<NDIM, DYN, 1>(p, pool, L); break;
                case 2: if constexpr (NDIM > 2) passA_stage1<NDIM, DYN, 2>(p, pool, L); break;
                case 3: if constexpr (NDIM > 3) passA_stage1<NDIM, DYN, 3>(p, pool, L); break;
                case 4: if constexpr (NDIM > 4) passA_stage1<NDIM, DYN, 4>(p, pool, L); break;
                case 5: if constexpr (NDIM > 5) passA_stage1<NDIM, DYN, 5>(p, pool, L); break;
            }
        }
        if (grp < GROUPS) sT[grp][j][lane] = L.T;
        __syncthreads();
        double part = 0.0;
        unsigned mask = 0;
        if (L.valid) {
            double S = 0.0;
#pragma unroll
            for (int l = 0; l < NDIM; ++l) S += sT[grp][l][lane];
            switch (j) {
                case 0: part = passA_stage2<0>(p, pool, L, S, mask); break;
                case 1: part = passA_stage2<1>(p, pool, L, S, mask); break;
                case 2: part = passA_stage2<2>(p, pool, L, S, mask); break;
                case 3: part = passA_stage2<3>(p, pool, L, S, mask); break;
                case 4: part = passA_stage2<4>(p, pool, L, S, mask); break;
                case 5: part = passA_stage2<5>(p, pool, L, S, mask); break;
            }
        }
        if (grp < GROUPS) { sPart[grp][j][lane] = part; sMask[grp][j][lane] = mask; }
        __syncthreads();
        if (L.valid && j == 0) {
            double acc = L.q0;
            unsigned m = 0;
#pragma unroll
            for (int l = 0; l < NDIM; ++l) { acc += sPart[grp][l][lane]; m |= sMask[grp][l][lane]; }
            pool.acc[L.i] = acc;
            pool.mask[L.i] = (uint16_t)m;
        }
    }
}

// ---- a5+a6 pass B: fetch the fluxes owned by neighbours, finish the update, sum the mass --------
template <int NDIM>
__device__ void phase_passB(const Params& p, const Pool& pool, DevState* st) {
    const uint32_t N = min(st->N, p.cap);
    const size_t cap = p.cap;
    double sum = 0.0;
    for (uint32_t i = gtid(); i < N; i += gthreads()) {
        double a = pool.acc[i];
        const unsigned mask = pool.mask[i];
#pragma unroll
        for (int j = 0; j < NDIM; ++j) {
            if (mask & (1u << j)) {          // lower face: flux computed by c-e^j as its upper face
                const uint32_t b = pool.nbr[(size_t)(2 * j) * cap + i];
                a += pool.phi[(size_t)(2 * j + 1) * cap + b];
            }
            if (mask & (1u << (8 + j))) {    // upper face: flux computed by c+e^j as its lower face
                const uint32_t b = pool.nbr[(size_t)(2 * j + 1) * cap + i];
                a -= pool.phi[(size_t)(2 * j) * cap + b];
            }
        }
        pool.Q[i] = a;
        sum += a;
    }
    sum = block_sum(sum);
    if (threadIdx.x == 0) pool.partial[blockIdx.x] = sum;
}

// plain sum of Q (init / correct / prune); same partial[] protocol as pass B
__device__ inline void phase_sum(const Params& p, const Pool& pool, DevState* st) {
    const uint32_t N = min(st->N, p.cap);
    double sum = 0.0;
    for (uint32_t i = gtid(); i < N; i += gthreads()) sum += pool.Q[i];
    sum = block_sum(sum);
    if (threadIdx.x == 0) pool.partial[blockIdx.x] = sum;
}

// one block: add the partials in index order, set the scale. after_step: advance t, count.
__device__ inline void finish_sum(const Params& p, const Pool& pool, DevState* st, unsigned nparts, bool after_step) {
    double v = 0.0;
    for (unsigned k = threadIdx.x; k < nparts; k += blockDim.x) v += pool.partial[k];
    v = block_sum(v);
    if (threadIdx.x == 0) {
        st->sumQ = v;
        if (!(v > 0.0) || !isfinite(v)) {
            if (p.normalise || !isfinite(v)) atomicOr(&st->err, E_DEGENERATE);
        }
        const double old = st->scale;
        st->mass = v * old;
        if (p.normalise && v > 0.0) st->scale = 1.0 / v;
        if (after_step) {
            const double dt = step_dt(p, st);
            if (!(dt > 0.0)) atomicOr(&st->err, E_DEGENERATE);
            st->dt = dt;
            st->t += dt;
            st->steps += 1;
            st->cell_updates += min(st->N, p.cap);
            st->inserted_total += min(st->N, p.cap) - st->N_before_grow;
        }
    }
}

}  // namespace gbees

namespace gbees {

// ---- a7 prune, D3 (Alg. 3) -------------------------------------------
// mark: keep c if P_c >= p*, and keep every existing grow-target of such a cell.
template <int NDIM, int DYN>
__device__ void phase_mark(const Params& p, const Pool& pool, DevState* st) {
    const uint32_t N = min(st->N, p.cap);
    const double scale = st->scale;
    const uint64_t slots = st->slots;
    for (uint32_t i = gtid(); i < N; i += gthreads()) {
        const uint64_t kf = pool.key[i];
        if (!(scale * pool.Q[i] >= p.thresh)) continue;
        pool.keep[i] = 1;
        const uint64_t key = kf & ~KEY_GROWN;
        int32_t c[NDIM];
        unpack<NDIM>(p, key, c);
        double ul[NDIM], uu[NDIM];
        face_velocities<NDIM, DYN>(p, c, ul, uu);
        for_each_target<NDIM>(p, key, c, ul, uu, [&](uint64_t tk, bool ok) {
            if (!ok) return;
            const uint32_t nb = ht_find(pool.table, slots, tk);
            if (nb != NBR_NONE) pool.keep[nb] = 1;
        });
    }
}

// Single-pass stream compaction with a decoupled-lookback scan over tiles of SCAN_TILE flags.
// tile_state[t] = (status << 32) | value, status 0 = invalid, 1 = aggregate, 2 = inclusive prefix.
// Tiles are handed out by an atomic counter so a tile's predecessors are always running or done.
constexpr int SCAN_ITEMS = 8;
constexpr int SCAN_TILE = TPB * SCAN_ITEMS;

// Generic core: flags -> stable destination index; body(i, dst) is called for kept items.
template <typename KeepFn, typename MoveFn, typename DropFn>
__device__ void scan_compact(uint32_t N, unsigned long long* tile_state, unsigned int* tile_counter,
                             uint32_t* total_out, KeepFn keepf, MoveFn movef, DropFn dropf) {
    __shared__ unsigned s_tile;
    __shared__ uint32_t s_warp[TPB / 32];
    __shared__ uint32_t s_prefix;
    const unsigned ntiles = (N + SCAN_TILE - 1) / SCAN_TILE;
    for (;;) {
        __syncthreads();
        if (threadIdx.x == 0) s_tile = atomicAdd(tile_counter, 1u);
        __syncthreads();
        const unsigned tile = s_tile;
        if (tile >= ntiles) break;
        const uint32_t base = tile * SCAN_TILE + threadIdx.x * SCAN_ITEMS;
        uint32_t f[SCAN_ITEMS], local = 0;
#pragma unroll
        for (int k = 0; k < SCAN_ITEMS; ++k) {
            f[k] = (base + k < N && keepf(base + k)) ? 1u : 0u;
            local += f[k];
        }
        // block exclusive scan of `local`
        uint32_t incl = local;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t v = __shfl_up_sync(0xffffffffu, incl, o);
            if ((threadIdx.x & 31) >= o) incl += v;
        }
        if ((threadIdx.x & 31) == 31) s_warp[threadIdx.x >> 5] = incl;
        __syncthreads();
        uint32_t woff = 0, tile_total = 0;
#pragma unroll
        for (int w = 0; w < TPB / 32; ++w) {
            if (w < (int)(threadIdx.x >> 5)) woff += s_warp[w];
            tile_total += s_warp[w];
        }
        // publish aggregate, look back
        if (threadIdx.x == 0) {
            if (tile == 0) {
                atomicExch(&tile_state[0], (2ull << 32) | tile_total);
                s_prefix = 0;
            } else {
                atomicExch(&tile_state[tile], (1ull << 32) | tile_total);
                uint32_t run = 0;
                for (int t = (int)tile - 1;; --t) {
                    unsigned long long v;
                    do { v = *reinterpret_cast<volatile unsigned long long*>(&tile_state[t]); } while ((v >> 32) == 0);
                    run += (uint32_t)v;
                    if ((v >> 32) == 2) break;
                }
                atomicExch(&tile_state[tile], (2ull << 32) | (run + tile_total));
                s_prefix = run;
            }
            if (tile == ntiles - 1) *total_out = s_prefix + tile_total;
        }
        __syncthreads();
        uint32_t dst = s_prefix + woff + (incl - local);
#pragma unroll
        for (int k = 0; k < SCAN_ITEMS; ++k) {
            if (f[k]) movef(base + k, dst++);
            else if (base + k < N) dropf(base + k);
        }
    }
}

__device__ inline void phase_compact(const Params& p, const Pool& pool, DevState* st) {
    const uint32_t N = min(st->N, p.cap);
    const double scale = st->scale;
    const double thresh = p.thresh;
    if (N == 0) { if (gtid() == 0) st->N_after_prune = 0; return; }
    scan_compact(
        N, pool.tile_state, &st->tile_counter, &st->N_after_prune,
        [&](uint32_t i) { return pool.keep[i] != 0; },
        [&](uint32_t i, uint32_t d) {
            const uint64_t kf = pool.key[i];
            const double q = pool.Q[i];
            // the GROWN flag survives only for cells still >= p* (their targets were all kept)
            pool.key2[d] = (scale * q >= thresh) ? kf : (kf & ~KEY_GROWN);
            pool.Q2[d] = q;
            pool.newidx[i] = d;
        },
        [&](uint32_t i) { pool.newidx[i] = NBR_NONE; });
}

// Adjacency after a prune, without touching the hashtable: old rows are translated through
// newidx. A pruned direct neighbour x is replaced by the tagged two-hop cell behind it (x's own
// direct neighbour in the same direction) if that one survives. Work item = (direction, old row).
__device__ inline void phase_remap(const Params& p, const Pool& pool, uint32_t N_old, int ndir) {
    const size_t cap = p.cap;
    const uint64_t items = (uint64_t)N_old * ndir;
    for (uint64_t w = gtid(); w < items; w += gthreads()) {
        const int d = (int)(w / N_old);
        const uint32_t i = (uint32_t)(w - (uint64_t)d * N_old);
        const uint32_t ni = pool.newidx[i];
        if (ni == NBR_NONE) continue;
        const uint32_t v = pool.nbr[(size_t)d * cap + i];
        uint32_t out = NBR_NONE;
        if (v != NBR_NONE) {
            if (v < NBR_TAG) {
                const uint32_t nv = pool.newidx[v];
                if (nv != NBR_NONE) out = nv;
                else {
                    const uint32_t y = pool.nbr[(size_t)d * cap + v];
                    if (y < NBR_TAG) {
                        const uint32_t ny = pool.newidx[y];
                        if (ny != NBR_NONE) out = NBR_TAG | ny;
                    }
                }
            } else {
                const uint32_t ny = pool.newidx[v & ~NBR_TAG];
                if (ny != NBR_NONE) out = NBR_TAG | ny;
            }
        }
        pool.nbr2[(size_t)d * cap + ni] = out;
    }
}

// clear the active part of the table (st->slots was set for the new cell count)
__device__ inline void phase_clear_table(const Pool& pool, const DevState* st) {
    const uint64_t slots = st->slots;
    const ulonglong2 e = make_ulonglong2(KEY_EMPTY, KEY_EMPTY);
    for (uint64_t s = gtid(); s < slots; s += gthreads()) pool.table[s] = e;
}

// CFL maximum over all cells (after a prune the running maximum must be recomputed)
template <int NDIM, int DYN>
__device__ void phase_smax(const Params& p, const Pool& pool, DevState* st) {
    const uint32_t N = min(st->N, p.cap);
    double smax = 0.0;
    for (uint32_t i = gtid(); i < N; i += gthreads()) {
        int32_t c[NDIM];
        unpack<NDIM>(p, pool.key[i] & ~KEY_GROWN, c);
        double ul[NDIM], uu[NDIM];
        face_velocities<NDIM, DYN>(p, c, ul, uu);
        smax = fmax(smax, cfl_term<NDIM>(p, ul));
    }
    smax = block_max(smax);
    if (threadIdx.x == 0 && smax > 0.0) atomicMax(&st->smax_bits, (unsigned long long)__double_as_longlong(smax));
}

// after the pointer swap: insert every pool key with its row index (table was cleared)
__device__ inline void phase_rebuild(const Params& p, const Pool& pool, DevState* st) {
    const uint32_t N = min(st->N, p.cap);
    const uint64_t slots = st->slots;
    for (uint32_t i = gtid(); i < N; i += gthreads()) {
        const uint64_t key = pool.key[i] & ~KEY_GROWN;
        const uint64_t s = ht_claim(pool.table, slots, key);
        if (s >= ~0ull - 1) { atomicOr(&st->err, s == ~0ull ? E_DEGENERATE : E_TABLE_FULL); continue; }  // duplicate key
        pool.table[s].y = i;
    }
}

// ---- D5 / A8 init_gaussian: one thread per candidate cell of the ellipsoid's bounding box ---------
struct GaussArgs {
    double inv[MAXN * MAXN];   // Sigma^-1 (or R^-1 for correct)
    double v[MAXN];            // correct: measurement z
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

template <int NDIM>
__device__ void phase_init_gaussian(const Params& p, const Pool& pool, DevState* st, const GaussArgs& g) {
    const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
    for (unsigned long long r = gtid(); r < g.total; r += stride) {
        int32_t c[NDIM];
        unsigned long long rem = r;
#pragma unroll
        for (int j = NDIM - 1; j >= 0; --j) {
            const unsigned long long w = 2ull * g.R[j] + 1ull;
            c[j] = (int32_t)((long long)(rem % w) - g.R[j]);
            rem /= w;
        }
        double d[NDIM];
#pragma unroll
        for (int j = 0; j < NDIM; ++j) d[j] = (double)c[j] * p.h[j];
        const double val = exp(-0.5 * quad_form<NDIM>(g.inv, d)) * g.norm;
        if (!(val >= p.thresh)) continue;
        bool ok = true;
#pragma unroll
        for (int j = 0; j < NDIM; ++j) ok = ok && c[j] >= -p.bias && c[j] <= p.bias - 1;
        if (!ok) { atomicOr(&st->err, E_KEY_RANGE); continue; }
        const uint32_t idx = atomicAdd(&st->N, 1u);
        if (idx >= p.cap) { atomicOr(&st->err, E_CAPACITY); continue; }
        pool.key[idx] = pack<NDIM>(p, c);
        pool.Q[idx] = val;
    }
}

// ---- a8 correct, D4 / Eq. (4): Q_c *= exp(-1/2 (z - x_c)^T R^-1 (z - x_c)) ------------
template <int NDIM>
__device__ void phase_correct(const Params& p, const Pool& pool, DevState* st, const GaussArgs& g) {
    const uint32_t N = min(st->N, p.cap);
    for (uint32_t i = gtid(); i < N; i += gthreads()) {
        int32_t c[NDIM];
        unpack<NDIM>(p, pool.key[i] & ~KEY_GROWN, c);
        double d[NDIM];
#pragma unroll
        for (int j = 0; j < NDIM; ++j) d[j] = g.v[j] - (p.mu[j] + (double)c[j] * p.h[j]);
        pool.Q[i] *= exp(-0.5 * quad_form<NDIM>(g.inv, d));
    }
}

template <int NDIM>
__device__ void phase_export(const Params& p, const Pool& pool, const DevState* st, int32_t* keys, double* out) {
    const uint32_t N = min(st->N, p.cap);
    const double scale = st->scale;
    for (uint32_t i = gtid(); i < N; i += gthreads()) {
        if (keys) {
            int32_t c[NDIM];
            unpack<NDIM>(p, pool.key[i] & ~KEY_GROWN, c);
#pragma unroll
            for (int j = 0; j < NDIM; ++j) keys[(size_t)i * NDIM + j] = c[j];
        }
        if (out) out[i] = scale * pool.Q[i];
    }
}

template <int NDIM>
__device__ void phase_import(const Params& p, const Pool& pool, DevState* st, const int32_t* keys,
                             const double* vals, uint32_t count) {
    for (uint32_t i = gtid(); i < count; i += gthreads()) {
        int32_t c[NDIM];
        bool ok = true;
#pragma unroll
        for (int j = 0; j < NDIM; ++j) {
            c[j] = keys[(size_t)i * NDIM + j];
            ok = ok && c[j] >= -p.bias && c[j] <= p.bias - 1;
        }
        if (!ok) { atomicOr(&st->err, E_KEY_RANGE); for (int j = 0; j < NDIM; ++j) c[j] = 0; }
        pool.key[i] = pack<NDIM>(p, c);
        pool.Q[i] = vals[i];
    }
}

}  // namespace gbees

#include <cooperative_groups.h>

namespace gbees {

struct RunArgs {
    double t_target;
    long long max_steps;
    int prune_every;
    int no_grow;
};

// pass B + mass sum + step bookkeeping without an extra barrier: the last block to finish (ticket)
// adds the per-block partials in index order (deterministic) and closes the step.
template <int NDIM>
__device__ void phase_passB_finish(const Params& p, const Pool& pool, DevState* st) {
    __shared__ bool s_last;
    phase_passB<NDIM>(p, pool, st);
    if (threadIdx.x == 0) {
        __threadfence();
        s_last = atomicAdd(&st->ticket, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (s_last) {
        __threadfence();
        finish_sum(p, pool, st, gridDim.x, true);
        if (threadIdx.x == 0) st->ticket = 0;
    }
}

// ---- a9 persistent cooperative step loop -----------------------------------------
// Same phases, same order and same arithmetic as gbees_step / gbees_prune; grid.sync() replaces the
// kernel boundaries. 4 barriers per step: grow | link | pass A | pass B + finish.
template <int NDIM, int DYN>
__device__ void phase_run(const Params& p, Pool pool, DevState* st, const RunArgs a) {
    namespace cg = cooperative_groups;
    cg::grid_group grid = cg::this_grid();
    long long k = 0;
    unsigned long long t_last = 0;
    if (gtid() == 0) asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t_last));
    // attribute the time since the previous tick (phase body + its barrier) to phase `ph`
    auto tick = [&](int ph) {
        if (gtid() == 0) {
            unsigned long long now;
            asm volatile("mov.u64 %0, %globaltimer;" : "=l"(now));
            st->phase_ns[ph] += now - t_last;
            t_last = now;
        }
    };
    for (;;) {
        // uniform decisions: every thread reads the same state after the barrier
        const double t = st->t;
        if (k >= a.max_steps || !(t < a.t_target) || st->err != 0) break;
        if (gtid() == 0) {
            st->N_before_grow = st->N;
            st->dt_cap = a.t_target < 1e299 ? a.t_target - t : 0.0;
        }
        grid.sync();
        if (!a.no_grow) {
            phase_grow<NDIM, DYN>(p, pool, st);
            grid.sync();
            tick(0);
            if (st->N != st->N_before_grow) {
                phase_link<NDIM, DYN, false>(p, pool, st);
                grid.sync();
                tick(1);
            }
        }
        phase_passA<NDIM, DYN>(p, pool, st);
        grid.sync();
        tick(2);
        phase_passB_finish<NDIM>(p, pool, st);
        grid.sync();
        tick(3);
        ++k;
        if (st->err != 0) break;
        const bool do_prune = a.prune_every > 0 && (k % a.prune_every) == 0;
        if (!do_prune) {
            // the grid outgrew the active table: rehash into a larger one
            if ((double)st->N > p.load_factor * (double)st->slots && st->slots < p.slots) {
                grid.sync();
                if (gtid() == 0) st->slots = table_slots_for(p, min(st->N, p.cap));
                grid.sync();
                phase_clear_table(pool, st);
                grid.sync();
                phase_rebuild(p, pool, st);
                grid.sync();
            }
            continue;
        }
        // ---- prune (D3) ----
        {
            const uint32_t N = min(st->N, p.cap);
            for (uint32_t i = gtid(); i < N; i += gthreads()) pool.keep[i] = 0;
            const uint32_t ntiles = (N + SCAN_TILE - 1) / SCAN_TILE + 1;
            for (uint32_t i = gtid(); i < ntiles; i += gthreads()) pool.tile_state[i] = 0ull;
            if (gtid() == 0) st->tile_counter = 0u;
        }
        grid.sync();
        phase_mark<NDIM, DYN>(p, pool, st);
        grid.sync();
        tick(4);
        phase_compact(p, pool, st);
        grid.sync();
        if (gtid() == 0) {
            st->prune_scanned += st->N;
            st->prunes += 1;
            st->N_before_grow = st->N;
            st->N = st->N_after_prune;
            st->slots = table_slots_for(p, st->N);
            st->smax_bits = 0ull;
            st->tile_counter = 0u;
            st->parity ^= 1u;
        }
        grid.sync();
        tick(5);
        phase_remap(p, pool, st->N_before_grow, 2 * NDIM);
        phase_clear_table(pool, st);
        grid.sync();
        tick(7);
        { uint64_t* tk = pool.key; pool.key = pool.key2; pool.key2 = tk; }
        { double* tq = pool.Q; pool.Q = pool.Q2; pool.Q2 = tq; }
        { uint32_t* tn = pool.nbr; pool.nbr = pool.nbr2; pool.nbr2 = tn; }
        phase_rebuild(p, pool, st);
        phase_smax<NDIM, DYN>(p, pool, st);
        phase_sum(p, pool, st);
        grid.sync();
        if (blockIdx.x == 0) finish_sum(p, pool, st, gridDim.x, false);
        grid.sync();
        tick(6);
        if (st->N == 0 || st->err != 0) break;
    }
}

}  // namespace gbees
