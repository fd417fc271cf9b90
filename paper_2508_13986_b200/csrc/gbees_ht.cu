// BASELINE config 4: the hashtable / stream-compaction device code of the prediction step,
// exposed on its own (bulk insert, lookup, delete + compaction + rebuild) with probe counters.
#include <cstdio>

#include "../../include/gbees.h"
#include "gbees_prims.cuh"

using namespace gbees;

struct gbees_ht {
    ulonglong2* table = nullptr;
    uint64_t slots = 0;
    uint32_t* count = nullptr;              // device: next pool index
    unsigned long long* probes = nullptr;   // device: probe accumulator
    unsigned long long* tile_state = nullptr;
    unsigned int* tile_counter = nullptr;
    uint32_t* total = nullptr;
    uint64_t* keys2 = nullptr;
    int64_t keys2_cap = 0, tiles_cap = 0;
    int device = 0;
    unsigned grid = 148 * 8;
};

__device__ __forceinline__ void add_probes(unsigned long long* acc, unsigned np) {
    unsigned long long v = np;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0) atomicAdd(acc, v);
}

__global__ void __launch_bounds__(TPB) k_ht_insert(ulonglong2* table, uint64_t slots, const uint64_t* keys, int64_t k,
                                                   uint32_t* count, uint32_t* idx_out, unsigned long long* probes,
                                                   int assign_rows) {
    unsigned np = 0;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t i = gtid(); i < k; i += stride) {
        const uint64_t s = ht_claim(table, slots, keys[i], &np);
        uint32_t idx = NBR_NONE;
        if (s < ~0ull - 1) {
            idx = assign_rows ? (uint32_t)i : atomicAdd(count, 1u);
            table[s].y = idx;
        }
        if (idx_out) idx_out[i] = idx;
    }
    add_probes(probes, np);
}

__global__ void __launch_bounds__(TPB) k_ht_lookup(const ulonglong2* table, uint64_t slots, const uint64_t* q, int64_t k,
                                                   uint32_t* out, unsigned long long* probes) {
    unsigned np = 0;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t i = gtid(); i < k; i += stride) {
        const uint32_t r = ht_find(table, slots, q[i], &np);
        if (out) out[i] = r;
    }
    add_probes(probes, np);
}

// Cooperative probing (north_star: "warp-cooperative probing"): a tile of W lanes serves one query and
// inspects W consecutive 16-byte slots per round (W = 4: 64 bytes = two sectors; W = 32: 512 bytes),
// so a long probe chain costs ceil(len / W) dependent memory rounds instead of len. The lanes of a
// tile take the tile's queries in turn (lane t of the tile owns query t). probes = slots up to and
// including the one that ended the search, as in the scalar kernel.
template <int W>
__global__ void __launch_bounds__(TPB) k_ht_lookup_coop(const ulonglong2* __restrict__ table, uint64_t slots, const uint64_t* q,
                                                        int64_t k, uint32_t* out, unsigned long long* probes) {
    const unsigned lane = threadIdx.x & 31, tl = lane % W, tbase = lane - tl;
    const unsigned tmask = (W == 32 ? 0xffffffffu : ((1u << W) - 1u) << tbase);
    unsigned np = 0;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    const int64_t kk = (k + stride - 1) / stride * stride;      // all lanes of a tile iterate together
    for (int64_t i = gtid(); i < kk; i += stride) {
        const bool have = i < k;
        const uint64_t myq = have ? q[i] : 0ull;
        uint32_t myres = NBR_NONE;
        for (int t = 0; t < W; ++t) {
            const uint64_t key = __shfl_sync(tmask, myq, tbase + t);
            const bool valid = __shfl_sync(tmask, (int)have, tbase + t) != 0;
            if (!valid) continue;                                 // uniform within the tile
            uint64_t s = home_slot(key, slots);
            uint32_t res = NBR_NONE;
            for (;;) {
                uint64_t ss = s + tl;
                if (ss >= slots) ss -= slots;
                const ulonglong2 e = table[ss];
                const unsigned hit = __ballot_sync(tmask, e.x == key) >> tbase;
                const unsigned emp = __ballot_sync(tmask, e.x == KEY_EMPTY) >> tbase;
                const unsigned ev = (hit | emp) & (W == 32 ? 0xffffffffu : (1u << W) - 1u);
                if (ev) {
                    const int first = __ffs((int)ev) - 1;
                    if ((hit >> first) & 1u) res = (uint32_t)__shfl_sync(tmask, (unsigned)e.y, tbase + first);
                    if ((int)tl == t) np += (unsigned)first + 1u;
                    break;
                }
                if ((int)tl == t) np += W;
                s += W;
                if (s >= slots) s -= slots;
            }
            if ((int)tl == t) myres = res;
        }
        if (have && out) out[i] = myres;
    }
    add_probes(probes, np);
}

__global__ void __launch_bounds__(TPB) k_ht_compact(const uint64_t* keys, const uint8_t* del, uint32_t k, uint64_t* keys2,
                                                    unsigned long long* tile_state, unsigned int* tile_counter,
                                                    uint32_t* total) {
    scan_compact(k, tile_state, tile_counter, total,
                 [&](uint32_t i) { return del[i] == 0; },
                 [&](uint32_t i, uint32_t d) { keys2[d] = keys[i]; },
                 [&](uint32_t) {});
}

#define HT_CU(call)                                                                    \
    do {                                                                               \
        cudaError_t e_ = (call);                                                       \
        if (e_ != cudaSuccess) {                                                       \
            fprintf(stderr, "gbees_ht: %s: %s\n", #call, cudaGetErrorString(e_));      \
            return GBEES_ERR_CUDA;                                                     \
        }                                                                              \
    } while (0)

extern "C" {

int gbees_ht_destroy(gbees_ht* h) {
    if (!h) return GBEES_OK;
    cudaSetDevice(h->device);
    cudaFree(h->table); cudaFree(h->count); cudaFree(h->probes); cudaFree(h->tile_state);
    cudaFree(h->tile_counter); cudaFree(h->total); cudaFree(h->keys2);
    delete h;
    return GBEES_OK;
}

int gbees_ht_create(gbees_ht** out, int64_t slots, int device) {
    if (!out || slots < 2) return GBEES_ERR_ARG;
    gbees_ht* h = new gbees_ht();
    h->device = device;
    h->slots = (uint64_t)slots;
    // on any failure the handle and whatever was allocated so far are released
    auto build = [&]() -> int {
        HT_CU(cudaSetDevice(device));
        cudaDeviceProp prop;
        HT_CU(cudaGetDeviceProperties(&prop, device));
        h->grid = (unsigned)prop.multiProcessorCount * 8u;
        HT_CU(cudaMalloc((void**)&h->table, h->slots * sizeof(ulonglong2)));
        HT_CU(cudaMalloc((void**)&h->count, 4));
        HT_CU(cudaMalloc((void**)&h->probes, 8));
        HT_CU(cudaMalloc((void**)&h->tile_counter, 4));
        HT_CU(cudaMalloc((void**)&h->total, 4));
        HT_CU(cudaMemset(h->table, 0xFF, h->slots * sizeof(ulonglong2)));
        HT_CU(cudaMemset(h->count, 0, 4));
        return GBEES_OK;
    };
    const int rc = build();
    if (rc != GBEES_OK) { gbees_ht_destroy(h); return rc; }
    *out = h;
    return GBEES_OK;
}

int gbees_ht_insert(gbees_ht* h, const uint64_t* keys, int64_t k, uint32_t* idx_out, uint64_t* probes) {
    if (!h || !keys || k < 0) return GBEES_ERR_ARG;
    HT_CU(cudaSetDevice(h->device));
    HT_CU(cudaMemset(h->probes, 0, 8));
    k_ht_insert<<<h->grid, TPB>>>(h->table, h->slots, keys, k, h->count, idx_out, h->probes, 0);
    HT_CU(cudaGetLastError());
    unsigned long long pr = 0;
    HT_CU(cudaMemcpy(&pr, h->probes, 8, cudaMemcpyDeviceToHost));
    if (probes) *probes = pr;
    return GBEES_OK;
}

int gbees_ht_lookup(gbees_ht* h, const uint64_t* q, int64_t k, uint32_t* out, uint64_t* probes) {
    if (!h || !q || k < 0) return GBEES_ERR_ARG;
    HT_CU(cudaSetDevice(h->device));
    HT_CU(cudaMemset(h->probes, 0, 8));
    k_ht_lookup<<<h->grid, TPB>>>(h->table, h->slots, q, k, out, h->probes);
    HT_CU(cudaGetLastError());
    unsigned long long pr = 0;
    HT_CU(cudaMemcpy(&pr, h->probes, 8, cudaMemcpyDeviceToHost));
    if (probes) *probes = pr;
    return GBEES_OK;
}

int gbees_ht_lookup_coop(gbees_ht* h, const uint64_t* q, int64_t k, uint32_t* out, uint64_t* probes, int width) {
    if (!h || !q || k < 0 || (width != 4 && width != 8 && width != 32)) return GBEES_ERR_ARG;
    HT_CU(cudaSetDevice(h->device));
    HT_CU(cudaMemset(h->probes, 0, 8));
    if (width == 4) k_ht_lookup_coop<4><<<h->grid, TPB>>>(h->table, h->slots, q, k, out, h->probes);
    else if (width == 8) k_ht_lookup_coop<8><<<h->grid, TPB>>>(h->table, h->slots, q, k, out, h->probes);
    else k_ht_lookup_coop<32><<<h->grid, TPB>>>(h->table, h->slots, q, k, out, h->probes);
    HT_CU(cudaGetLastError());
    unsigned long long pr = 0;
    HT_CU(cudaMemcpy(&pr, h->probes, 8, cudaMemcpyDeviceToHost));
    if (probes) *probes = pr;
    return GBEES_OK;
}

int gbees_ht_compact(gbees_ht* h, uint64_t* keys, const uint8_t* del, int64_t k, int64_t* k_out) {
    if (!h || !keys || !del || k < 0 || k >= (int64_t)0x80000000u) return GBEES_ERR_ARG;
    HT_CU(cudaSetDevice(h->device));
    const int64_t tiles = (k + SCAN_TILE - 1) / SCAN_TILE + 1;
    if (k > h->keys2_cap) { cudaFree(h->keys2); HT_CU(cudaMalloc((void**)&h->keys2, (size_t)k * 8)); h->keys2_cap = k; }
    if (tiles > h->tiles_cap) { cudaFree(h->tile_state); HT_CU(cudaMalloc((void**)&h->tile_state, (size_t)tiles * 8)); h->tiles_cap = tiles; }
    HT_CU(cudaMemsetAsync(h->tile_state, 0, (size_t)tiles * 8));
    HT_CU(cudaMemsetAsync(h->tile_counter, 0, 4));
    HT_CU(cudaMemsetAsync(h->total, 0, 4));
    if (k > 0) k_ht_compact<<<h->grid, TPB>>>(keys, del, (uint32_t)k, h->keys2, h->tile_state, h->tile_counter, h->total);
    uint32_t kept = 0;
    HT_CU(cudaMemcpy(&kept, h->total, 4, cudaMemcpyDeviceToHost));
    HT_CU(cudaMemcpyAsync(keys, h->keys2, (size_t)kept * 8, cudaMemcpyDeviceToDevice));
    HT_CU(cudaMemsetAsync(h->table, 0xFF, h->slots * sizeof(ulonglong2)));
    HT_CU(cudaMemsetAsync(h->probes, 0, 8));
    k_ht_insert<<<h->grid, TPB>>>(h->table, h->slots, keys, kept, h->count, nullptr, h->probes, 1);
    HT_CU(cudaMemcpyAsync(h->count, &kept, 4, cudaMemcpyHostToDevice));
    HT_CU(cudaDeviceSynchronize());
    if (k_out) *k_out = kept;
    return GBEES_OK;
}

}  // extern "C"
