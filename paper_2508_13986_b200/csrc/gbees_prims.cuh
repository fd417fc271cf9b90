// Parallel primitives shared by the prediction-step kernels and the config-4 hashtable microbench:
// warp/block reductions (here warp shuffles + one block stage) and a single-pass
// decoupled-lookback scan for stream compaction (PAPER.md:291 describes a two-stage scan).
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

}  // namespace gbees
