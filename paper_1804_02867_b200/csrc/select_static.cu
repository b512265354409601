// efm_beam_threshold_static(): the beam threshold selection (a-4) for callers that have no way to get
// device memory for its scratch.
//
// Who that is.  Everything else in this library works inside ONE workspace the caller allocated; that suits a program
// that owns its GPU.  It does not suit code that is a guest on somebody else's GPU: a step that runs inside a host
// application (a solver plug-in, a serving process, a job under a memory-capped scheduler) whose allocator has already
// handed out all of HBM and gives a guest nothing, or a latency-bound loop where cudaMalloc / cudaFree are banned
// because both may stall every stream of the device.  Such a caller can still pass its key array and an 8-byte result
// slot.  What it cannot supply is the scratch of the selection (2048-bin histogram, rank / prefix words, the compact
// key buffer).  Here that scratch is part of the library image: a file-scope __device__ array, EFM_STATIC_SELECT_BYTES
// (8 MiB + 8448 B) on every GPU that loads this module, held until the process exits.  Hence the limit of
// EFM_STATIC_SELECT_MAX_KEYS = 2^20 key slots per call, one level of a small beam; larger levels need
// efm_beam_threshold() / efm_enumerate() and a workspace.
//
// The kernels are the two-histogram + narrow selection of post.cu (k_select_hist x2, k_select_narrow) restated over a
// small control record; they also count the selectable keys themselves, since a caller outside the traversal has no
// LevelCtl that would know that number.
#include <cstdio>
#include <mutex>

#include "../../include/efm_b200.h"
#include "device_common.cuh"

namespace efm {
namespace {

constexpr int kThreads = 256;
constexpr int kTopBits = 11;                         // two 11-bit rounds over the caller's keys, then 42 bits on the compact copy
constexpr u64 kMaxKeys = EFM_STATIC_SELECT_MAX_KEYS;

struct StaticSel {
    u32 hist[SEL_BINS];        // must be zero when a call starts (cleared by the call itself, and again by the last block of a round)
    u64 prefix, rank, n_compact;
    u32 ticket, binds;         // binds: more than cap selectable keys, a threshold has to be found
    u64 pad[28];               // header = 8448 bytes = 33 * 256: ckeys stays 256-byte aligned
    u64 ckeys[kMaxKeys];       // keys that carry the selected 22-bit prefix; only [0, n_compact) is ever read
};
static_assert(sizeof(StaticSel) == EFM_STATIC_SELECT_BYTES, "header states the size of the built-in scratch");
constexpr size_t kHeaderBytes = sizeof(StaticSel) - sizeof(u64) * kMaxKeys;

// THE scratch.  In host code this name is only a stand-in for the symbol (taking its address there yields a host address a
// kernel must never see); the device address comes from cudaGetSymbolAddress() in static_select_setup() below.
static __device__ __align__(256) unsigned char g_static_select_scratch[sizeof(StaticSel)];

// Whole block: the bin b with cum(b) <= rank < cum(b) + h[b] and the sum of all bins.
__device__ void find_rank_bin(const u32* h, int nb, u64 rank, u32* s_bin, u64* s_cum, u64* s_total, u64* part) {
    const int T = blockDim.x, per = (nb + T - 1) / T, b0 = threadIdx.x * per;
    u64 sum = 0;
    for (int j = 0; j < per; ++j) if (b0 + j < nb) sum += h[b0 + j];
    part[threadIdx.x] = sum;
    if (threadIdx.x == 0) { *s_bin = (u32)(nb - 1); *s_cum = 0; }
    __syncthreads();
    for (int off = 1; off < T; off <<= 1) {
        const u64 v = threadIdx.x >= off ? part[threadIdx.x - off] : 0;
        __syncthreads();
        part[threadIdx.x] += v;
        __syncthreads();
    }
    const u64 incl = part[threadIdx.x];
    if (threadIdx.x == T - 1) *s_total = incl;
    u64 cum = incl - sum;
    if (cum <= rank && rank < incl)
        for (int j = 0; j < per; ++j) {
            const u64 c = h[b0 + j];
            if (rank < cum + c) { *s_bin = (u32)(b0 + j); *s_cum = cum; break; }
            cum += c;
        }
    __syncthreads();
}

// LEVEL 0: histogram of the top 11 bits of every selectable key (key < kKeyDone); the last block decides whether the beam
// binds at all (more than cap such keys) and, if so, which bin holds sorted position cap.  LEVEL 1: the next 11 bits of the
// keys inside that bin.
template <int LEVEL>
__global__ void __launch_bounds__(kThreads) k_static_select_hist(const u64* __restrict__ keys, u64 n, u64 cap, StaticSel* sel,
                                                                 u64* __restrict__ out) {
    if (LEVEL == 1 && !sel->binds) return;
    __shared__ u32 h[SEL_BINS];
    __shared__ u64 part[kThreads];
    __shared__ u32 s_bin; __shared__ u64 s_cum, s_total; __shared__ bool is_last;
    for (int b = threadIdx.x; b < SEL_BINS; b += kThreads) h[b] = 0;
    __syncthreads();
    const u64 top = LEVEL == 0 ? 0ULL : sel->prefix;
    constexpr int shift = 64 - kTopBits * (LEVEL + 1);
    for (u64 i = (u64)blockIdx.x * kThreads + threadIdx.x; i < n; i += (u64)gridDim.x * kThreads) {
        const u64 key = keys[i];
        if (key >= kKeyDone) continue;   // balanced child / unused slot: outside the ranking, as in the traversal
        if (LEVEL == 1 && (key >> (64 - kTopBits)) != top) continue;
        atomicAdd(&h[(u32)(key >> shift) & (u32)(SEL_BINS - 1)], 1u);
    }
    __syncthreads();
    for (int b = threadIdx.x; b < SEL_BINS; b += kThreads) if (h[b]) atomicAdd(&sel->hist[b], h[b]);
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) is_last = atomicAdd(&sel->ticket, 1u) == gridDim.x - 1;
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    for (int b = threadIdx.x; b < SEL_BINS; b += kThreads) { h[b] = ((volatile u32*)sel->hist)[b]; sel->hist[b] = 0; }
    __syncthreads();
    const u64 rank = LEVEL == 0 ? cap : sel->rank;
    find_rank_bin(h, SEL_BINS, rank, &s_bin, &s_cum, &s_total, part);
    if (threadIdx.x == 0) {
        sel->ticket = 0;
        if (LEVEL == 0 && s_total <= cap) { sel->binds = 0; *out = kKeySentinel; return; }   // everything is kept
        sel->binds = 1;
        sel->prefix = (LEVEL == 0 ? 0ULL : top << kTopBits) | s_bin;
        sel->rank = rank - s_cum;
        sel->n_compact = 0;
    }
}

// Copies the keys with the selected 22-bit prefix into the compact buffer; the last block settles the remaining 42 bits on
// that buffer alone (11 / 11 / 10 / 10-bit rounds in shared memory) and writes the threshold.
__global__ void __launch_bounds__(kThreads) k_static_select_narrow(const u64* __restrict__ keys, u64 n, StaticSel* sel, u64* __restrict__ out) {
    if (!sel->binds) return;
    __shared__ u32 h[SEL_BINS];
    __shared__ u64 part[kThreads];
    __shared__ u32 s_bin; __shared__ u64 s_cum, s_total; __shared__ bool is_last;
    const u64 top = sel->prefix;
    constexpr int kLow = 64 - 2 * kTopBits;
    const int lane = threadIdx.x & 31;
    for (u64 base = (u64)blockIdx.x * kThreads; base < n; base += (u64)gridDim.x * kThreads) {   // warp-uniform trip count
        const u64 i = base + threadIdx.x;
        const u64 key = i < n ? keys[i] : kKeySentinel;
        const bool hit = key < kKeyDone && (key >> kLow) == top;
        const u32 m = __ballot_sync(0xffffffffu, hit);
        if (m) {
            u64 pos = 0;
            if (lane == 0) pos = atomicAdd(&sel->n_compact, (u64)__popc(m));
            pos = __shfl_sync(0xffffffffu, pos, 0);
            if (hit && pos + __popc(m) <= kMaxKeys) sel->ckeys[pos + __popc(m & ((1u << lane) - 1u))] = key;   // n <= kMaxKeys: always true
        }
    }
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) is_last = atomicAdd(&sel->ticket, 1u) == gridDim.x - 1;
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    const u64 nc = min(*(volatile u64*)&sel->n_compact, kMaxKeys);
    u64 rank = sel->rank, prefix = 0;
    const int bits[4] = {11, 11, 10, 10};
    int shift = kLow;
    for (int r = 0; r < 4; ++r) {
        shift -= bits[r];
        const int nb = 1 << bits[r];
        for (int b = threadIdx.x; b < nb; b += kThreads) h[b] = 0;
        __syncthreads();
        const u64 low = (1ULL << kLow) - 1ULL;
        for (u64 i = threadIdx.x; i < nc; i += kThreads) {
            const u64 key = __ldcg(&sel->ckeys[i]) & low;
            if (r == 0 || (key >> (shift + bits[r])) == prefix) atomicAdd(&h[(key >> shift) & (u64)(nb - 1)], 1u);
        }
        __syncthreads();
        find_rank_bin(h, nb, rank, &s_bin, &s_cum, &s_total, part);
        prefix = (prefix << bits[r]) | (u64)s_bin;
        rank -= s_cum;
        __syncthreads();
    }
    if (threadIdx.x == 0) { *out = (top << kLow) | prefix; sel->ticket = 0; }
}

// ---- host side ------------------------------------------------------------------------------------------------------
constexpr int kMaxDevices = 64;
std::mutex g_mu;
StaticSel* g_scratch_ptr[kMaxDevices] = {};   // device address of g_static_select_scratch ON that device
int g_sm_count[kMaxDevices] = {};
thread_local char t_error[256] = "";

// Once per device, with that device current: ask the runtime where the array lives there.  Every GPU holds its own copy
// of a __device__ variable, so the address is looked up (and kept) per device ordinal.
int static_select_setup(int device, StaticSel** sel, int* sm_count) {
    std::lock_guard<std::mutex> lk(g_mu);
    if (!g_scratch_ptr[device]) {
        void* p = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&p, g_static_select_scratch);
        if (e == cudaSuccess && !p) e = cudaErrorInvalidSymbol;
        int sms = 0;
        if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
        if (e != cudaSuccess) {
            snprintf(t_error, sizeof t_error, "set-up of the built-in scratch on device %d: %s", device, cudaGetErrorString(e));
            cudaGetLastError();
            return EFM_E_CUDA;
        }
        g_scratch_ptr[device] = (StaticSel*)p;
        g_sm_count[device] = sms > 0 ? sms : 1;
    }
    *sel = g_scratch_ptr[device];
    *sm_count = g_sm_count[device];
    return EFM_OK;
}

}  // namespace
}  // namespace efm

using namespace efm;

extern "C" {

int efm_beam_threshold_static(const uint64_t* d_keys, int64_t n_keys, int64_t cap, uint64_t* d_threshold, int32_t device,
                              void* cuda_stream) {
    t_error[0] = 0;
    // argument checks first, before any CUDA call: the size limit is reported the same way on a box without a GPU
    if ((u64)(n_keys < 0 ? 0 : n_keys) > kMaxKeys) {
        snprintf(t_error, sizeof t_error,
                 "n_keys = %lld is more than EFM_STATIC_SELECT_MAX_KEYS = %llu, the size the built-in scratch array was compiled "
                 "for; use efm_beam_threshold() with caller-provided scratch",
                 (long long)n_keys, kMaxKeys);
        return EFM_E_CAPACITY;
    }
    if (n_keys < 0 || cap <= 0 || !d_threshold || (n_keys > 0 && !d_keys) || device < 0 || device >= kMaxDevices) {
        snprintf(t_error, sizeof t_error, "bad argument (n_keys %lld, cap %lld, device %d, or a NULL pointer)", (long long)n_keys,
                 (long long)cap, (int)device);
        return EFM_E_INVAL;
    }
    cudaError_t e = cudaSetDevice(device);
    if (e != cudaSuccess) {
        snprintf(t_error, sizeof t_error, "cudaSetDevice(%d): %s", (int)device, cudaGetErrorString(e));
        cudaGetLastError();
        return EFM_E_CUDA;
    }
    StaticSel* sel = nullptr;
    int sms = 1;
    const int rc = static_select_setup(device, &sel, &sms);
    if (rc != EFM_OK) return rc;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    // the array still holds what the previous call left: histogram, ticket and counters have to start at zero
    e = cudaMemsetAsync(sel, 0, kHeaderBytes, s);
    if (e == cudaSuccess) {
        u64 blocks = ((u64)n_keys + kThreads * 8 - 1) / (kThreads * 8);
        if (blocks > (u64)sms * 8) blocks = (u64)sms * 8;
        if (blocks < 1) blocks = 1;
        const u64* keys = (const u64*)d_keys;
        u64* out = (u64*)d_threshold;
        k_static_select_hist<0><<<(unsigned)blocks, kThreads, 0, s>>>(keys, (u64)n_keys, (u64)cap, sel, out);
        k_static_select_hist<1><<<(unsigned)blocks, kThreads, 0, s>>>(keys, (u64)n_keys, (u64)cap, sel, out);
        k_static_select_narrow<<<(unsigned)blocks, kThreads, 0, s>>>(keys, (u64)n_keys, sel, out);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) {
        snprintf(t_error, sizeof t_error, "launch: %s", cudaGetErrorString(e));
        return EFM_E_CUDA;
    }
    return EFM_OK;
}

const char* efm_beam_threshold_static_error(void) { return t_error; }

}  // extern "C"
