// gbees_marginal_noalloc: the marginal of a grid PDF for callers that cannot allocate --
// code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc. Same hash-accumulation
// as gbees_marginal (gbees_brick.cuh: phase_marg_*), but over an EXPORTED state (keys + masses in caller memory)
// and with its scratch table in a file-scope device array instead of a context's allocations.
//
// The scratch array is one per GPU that loads the library (held until the process exits), shared by every call
// and never cleared behind the caller's back: each call clears the part it uses first. Calls that overlap on the
// GPU (two streams, two threads) race on it. This file calls no cudaMalloc / cudaFree / allocating library routine.
#include <cstdio>
#include <mutex>
#include <string>

#include "../../include/gbees.h"
#include "gbees_prims.cuh"

using namespace gbees;

namespace {

constexpr unsigned long long NA_SLOTS = GBEES_NOALLOC_MAX_CELLS * 2ull;   // table slots at load factor <= 0.5
constexpr int NA_HDR = 32;                                                // header words: [0] output count, [1] error bits
// [header | slot keys (packed kept coordinates, KEY_EMPTY = free) | slot values (mass, as double bits)]: 4 MiB + 256 B
static __device__ __align__(256) unsigned long long g_na_scratch[NA_HDR + 2 * NA_SLOTS];

// In host code g_na_scratch is only a stand-in for the symbol, not a device address: the kernels get the address
// that cudaGetSymbolAddress reports, looked up once per device with that device current.
constexpr int NA_MAX_DEVICES = 64;
unsigned long long* g_na_ptr[NA_MAX_DEVICES] = {nullptr};
std::mutex g_na_mutex;
thread_local std::string g_na_error;

int na_fail(int code, const std::string& msg) {
    g_na_error = msg;
    fprintf(stderr, "gbees_marginal_noalloc: %s\n", msg.c_str());
    return code;
}

struct NaArgs {
    int n, m, mbits;
    int dims[MAXN];
    unsigned long long S;   // slots used by this call (power of two, <= NA_SLOTS)
};

__global__ void __launch_bounds__(TPB) k_na_clear(unsigned long long* scratch, unsigned long long S) {
    unsigned long long* skey = scratch + NA_HDR;
    unsigned long long* sval = skey + NA_SLOTS;
    if (gtid() < NA_HDR) scratch[gtid()] = 0ull;
    for (unsigned long long i = gtid(); i < S; i += gthreads()) { skey[i] = KEY_EMPTY; sval[i] = 0ull; }
}

__global__ void __launch_bounds__(TPB) k_na_accumulate(const __grid_constant__ NaArgs g, const int32_t* __restrict__ keys,
                                                       const double* __restrict__ p, unsigned long long N,
                                                       unsigned long long* scratch) {
    unsigned long long* skey = scratch + NA_HDR;
    double* sval = reinterpret_cast<double*>(skey + NA_SLOTS);
    int* err = reinterpret_cast<int*>(scratch + 1);
    const long long mbias = 1ll << (g.mbits - 1);
    for (unsigned long long i = gtid(); i < N; i += gthreads()) {
        unsigned long long key = 0ull;
        bool ok = true;
        for (int r = 0; r < g.m; ++r) {
            const long long cv = keys[i * g.n + g.dims[r]];
            ok = ok && cv >= -mbias && cv < mbias;
            key = (key << g.mbits) | (unsigned long long)(cv + mbias);
        }
        if (!ok) { atomicOr(err, E_KEY_RANGE); continue; }
        unsigned long long s = home_slot(key, g.S);
        for (unsigned long long tries = 0;; ++tries) {
            if (tries == g.S) { atomicOr(err, E_TABLE_FULL); break; }
            unsigned long long cur = *reinterpret_cast<volatile unsigned long long*>(&skey[s]);
            if (cur == KEY_EMPTY) cur = atomicCAS(&skey[s], KEY_EMPTY, key);
            if (cur == KEY_EMPTY || cur == key) { atomicAdd(&sval[s], p[i]); break; }
            if (++s == g.S) s = 0;
        }
    }
}

__global__ void __launch_bounds__(TPB) k_na_emit(const __grid_constant__ NaArgs g, unsigned long long* scratch,
                                                 int32_t* out_keys, double* out_p, unsigned long long cap) {
    const unsigned long long* skey = scratch + NA_HDR;
    const double* sval = reinterpret_cast<const double*>(skey + NA_SLOTS);
    const long long mbias = 1ll << (g.mbits - 1);
    const unsigned long long fm = g.mbits >= 64 ? ~0ull : (1ull << g.mbits) - 1ull;
    for (unsigned long long i = gtid(); i < g.S; i += gthreads()) {
        const unsigned long long key = skey[i];
        if (key == KEY_EMPTY) continue;
        const unsigned long long o = atomicAdd(&scratch[0], 1ull);
        if (o >= cap) continue;
        for (int r = 0; r < g.m; ++r)
            out_keys[o * g.m + r] = (int32_t)((long long)((key >> ((g.m - 1 - r) * g.mbits)) & fm) - mbias);
        out_p[o] = sval[i];
    }
}

// device address of the scratch array on `device` (which must be current), looked up once per device
int na_scratch(int device, unsigned long long** out) {
    if (device < 0 || device >= NA_MAX_DEVICES) return na_fail(GBEES_ERR_ARG, "device ordinal out of range");
    std::lock_guard<std::mutex> lock(g_na_mutex);
    if (!g_na_ptr[device]) {
        unsigned long long* ptr = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void**)&ptr, g_na_scratch);
        if (e != cudaSuccess || !ptr)
            return na_fail(GBEES_ERR_CUDA, std::string("cudaGetSymbolAddress(g_na_scratch): ") + cudaGetErrorString(e));
        g_na_ptr[device] = ptr;
    }
    *out = g_na_ptr[device];
    return GBEES_OK;
}

}  // namespace

extern "C" {

const char* gbees_marginal_noalloc_error(void) { return g_na_error.c_str(); }

int gbees_marginal_noalloc(int device, void* stream, int n, const int32_t* keys, const double* p, int64_t count_in,
                           const int* dims, int m, int32_t* out_keys, double* out_p, int64_t cap, int64_t* count) {
    if (!keys || !p || !dims || !out_keys || !out_p || !count || n < 1 || n > MAXN || m < 1 || m > n || count_in < 0 || cap < 0)
        return na_fail(GBEES_ERR_ARG, "bad argument");
    if (count_in > (int64_t)GBEES_NOALLOC_MAX_CELLS)
        return na_fail(GBEES_ERR_CAPACITY, "more than GBEES_NOALLOC_MAX_CELLS (" + std::to_string(GBEES_NOALLOC_MAX_CELLS) +
                                               ") input cells: the static scratch table cannot hold them; use gbees_marginal");
    NaArgs g;
    g.n = n; g.m = m;
    g.mbits = 63 / m > 32 ? 32 : 63 / m;
    for (int r = 0; r < MAXN; ++r) g.dims[r] = 0;
    for (int r = 0; r < m; ++r) {
        if (dims[r] < 0 || dims[r] >= n) return na_fail(GBEES_ERR_ARG, "dims entry out of [0, n)");
        for (int q = 0; q < r; ++q) if (dims[q] == dims[r]) return na_fail(GBEES_ERR_ARG, "dims entries must be distinct");
        g.dims[r] = dims[r];
    }
    *count = 0;
    if (count_in == 0) return GBEES_OK;
    cudaError_t e = cudaSetDevice(device);
    if (e != cudaSuccess) return na_fail(GBEES_ERR_CUDA, std::string("cudaSetDevice: ") + cudaGetErrorString(e));
    unsigned long long* scratch = nullptr;
    const int rc = na_scratch(device, &scratch);
    if (rc) return rc;
    g.S = 1024;
    while (g.S < 2ull * (unsigned long long)count_in) g.S <<= 1;      // at most N marginal cells: load factor <= 0.5
    cudaStream_t st = (cudaStream_t)stream;
    const unsigned grid = 148 * 4;
    k_na_clear<<<grid, TPB, 0, st>>>(scratch, g.S);                   // the array keeps the last call's contents
    k_na_accumulate<<<grid, TPB, 0, st>>>(g, keys, p, (unsigned long long)count_in, scratch);
    k_na_emit<<<grid, TPB, 0, st>>>(g, scratch, out_keys, out_p, (unsigned long long)cap);
    if ((e = cudaGetLastError()) != cudaSuccess) return na_fail(GBEES_ERR_CUDA, std::string("launch: ") + cudaGetErrorString(e));
    unsigned long long hdr[2] = {0ull, 0ull};
    if ((e = cudaMemcpyAsync(hdr, scratch, sizeof(hdr), cudaMemcpyDeviceToHost, st)) != cudaSuccess ||
        (e = cudaStreamSynchronize(st)) != cudaSuccess)
        return na_fail(GBEES_ERR_CUDA, std::string("read-back: ") + cudaGetErrorString(e));
    const int err = (int)(hdr[1] & 0xffffffffull);
    if (err & E_KEY_RANGE) return na_fail(GBEES_ERR_KEY_RANGE, "a kept coordinate does not fit floor(63/m) bits");
    if (err & E_TABLE_FULL) return na_fail(GBEES_ERR_CAPACITY, "scratch table full");
    *count = (int64_t)hdr[0];
    if (cap < *count) return na_fail(GBEES_ERR_BUFFER, "output buffers smaller than the marginal: *count rows are needed");
    return GBEES_OK;
}

}  // extern "C"
