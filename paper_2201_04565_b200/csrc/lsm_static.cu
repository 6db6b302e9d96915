// lsm_static.cu -- lsm_spring_energy_static: the elastic energy of a spring list (Eq. 1) for callers that
// cannot allocate device memory.
//
// Who those callers are.  Everything else in this library hangs off an lsm_sim handle, and lsm_create builds that handle
// with dozens of device allocations (cudaMalloc, or the caller's allocator callback).  Some users of the library hold the
// particle and spring arrays on the GPU already and want one number out of them -- the energy the paper plots in Fig. 4B
// -- from a place where asking the CUDA runtime for memory is not an option:
//   * an analysis step inside a simulation loop whose GPU memory was all handed to one arena or framework pool when the
//     process started (a 180 GB state of the config-5 kind is sized that way): a cudaMalloc there fails, or succeeds only
//     by taking memory the arena's owner counted on;
//   * a monitor that runs beside asynchronous lsm_step work: cudaFree waits for the whole device and cudaMalloc may, so
//     an allocation per sample stalls the step pipeline the rest of the library keeps asynchronous;
//   * code with a fixed memory budget that must be known when the library is loaded (long unattended parameter sweeps, the
//     paper's "high-throughput" use), where an out-of-memory failure hours in is not acceptable.
// For them this file keeps the one piece of scratch the computation needs -- the per-block partial sums of the deterministic
// two-level reduction, the same scheme as k_reduce_chunks / k_finalize_sample in lsm_kernels.cuh -- in a file-scope
// __device__ array of fixed size instead of an allocation.  The price: every GPU that loads liblsm_b200.so carries those
// 524,544 bytes until the process exits, the spring list is limited to LSM_STATIC_MAX_SPRINGS, and all calls on one
// device share the one array (see the header).
//
// This file shares no state with lsm_api.cu and changes nothing there.  It calls no cudaMalloc, cudaFree, or library
// routine that allocates; host-side it uses a fixed table and the caller's error buffer only.
#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <mutex>

#include "../../include/lsm.h"

namespace {

constexpr int kSBlock = 1024;                    // threads per block: short threads (8 springs each), 64 warps per SM in flight --
                                                 // the loop is three dependent loads deep (flag -> ids -> positions), so it
                                                 // is latency-bound: 256 threads x 32 springs took 114 us on config 3 (measured)
constexpr int kSPerThread = 8;                   // springs per thread
constexpr int kSChunk = kSBlock * kSPerThread;   // 8192 springs per block, a fixed cut: the summation order does not depend on the GPU
constexpr long long kSMaxBlocks = LSM_STATIC_MAX_SPRINGS / kSChunk;   // 32768
static_assert(kSMaxBlocks * kSChunk == LSM_STATIC_MAX_SPRINGS, "the maximum is a whole number of blocks");

// Layout of the static scratch (bytes): [0, 256) header, word 0 = springs skipped for bad endpoint ids (must be zero when
// the first kernel starts: cleared by a cudaMemsetAsync in front of it); then kSMaxBlocks partial energies (double); then
// kSMaxBlocks partial counts of live springs (uint64).  The partials need no clearing: the first kernel of a call writes
// every entry the second one reads, entries past this call's block count keep older values and are never read.
constexpr size_t kSHeaderBytes = 256;
constexpr size_t kSScratchBytes = kSHeaderBytes + (size_t)kSMaxBlocks * 16;

// In host code this name is only a handle for cudaGetSymbolAddress: it is NOT a device address and must never be passed
// to a kernel.  Device code below may name it directly; the kernels take the looked-up pointer instead so that there is
// one way of reaching the memory.
static __device__ __align__(256) unsigned char g_static_scratch[kSScratchBytes];

struct StaticView {
    unsigned long long *bad;       // [1]
    double *partU;                 // [kSMaxBlocks]
    unsigned long long *partN;     // [kSMaxBlocks]
};

__device__ __forceinline__ StaticView view_of(unsigned char *base) {
    StaticView v;
    v.bad = reinterpret_cast<unsigned long long *>(base);
    v.partU = reinterpret_cast<double *>(base + kSHeaderBytes);
    v.partN = reinterpret_cast<unsigned long long *>(base + kSHeaderBytes + (size_t)kSMaxBlocks * 8);
    return v;
}

struct EnergyArgs {
    const double *x;               // [N*dim] interleaved
    const int32_t *si, *sj;        // [M]
    const double *k, *r0;          // [M] or NULL -> uniform
    const uint8_t *broken;         // [M] or NULL
    double k_u, r0_u;
    long long N, M;
};

__device__ __forceinline__ double warp_sum_d(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Fixed-order block sum: xor-shuffle tree inside each warp, then the 32 warp sums in warp order (every thread gets it).
__device__ __forceinline__ double block_sum_d(double v, double *sh8) {
    v = warp_sum_d(v);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) sh8[threadIdx.x >> 5] = v;
    __syncthreads();
    double t = 0.0;
#pragma unroll
    for (int w = 0; w < kSBlock / 32; ++w) t += sh8[w];
    return t;
}

__device__ __forceinline__ unsigned long long block_sum_u(unsigned long long v, unsigned long long *sh8) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) sh8[threadIdx.x >> 5] = v;
    __syncthreads();
    unsigned long long t = 0;
#pragma unroll
    for (int w = 0; w < kSBlock / 32; ++w) t += sh8[w];
    return t;
}

// Level 1: block c sums the springs [c * 8192, (c + 1) * 8192): thread t takes c * 8192 + i * 1024 + t for i = 0 .. 7 in
// that order (coalesced list reads, two gathered positions per spring), u = k (r - r0)^2 / 2 with an IEEE square root.
// A broken spring contributes nothing (the (1 - Xi) factor of Eq. 1, kept irreversible by the caller's flag array as in
// PAPER.md:L98, L196); a spring with an endpoint outside [0, N) or with i == j is skipped and counted.
template <int D>
__global__ void __launch_bounds__(kSBlock) k_static_energy_partials(const EnergyArgs A, unsigned char *scratch) {
    __shared__ double shd[kSBlock / 32];
    __shared__ unsigned long long shu[kSBlock / 32];
    const StaticView S = view_of(scratch);
    const long long base = (long long)blockIdx.x * kSChunk;
    double u = 0.0;
    unsigned long long live = 0, bad = 0;
#pragma unroll 4
    for (int it = 0; it < kSPerThread; ++it) {
        const long long s = base + (long long)it * kSBlock + threadIdx.x;
        if (s >= A.M) break;
        if (A.broken && A.broken[s]) continue;
        const long long i = A.si[s], j = A.sj[s];
        if (i < 0 || j < 0 || i >= A.N || j >= A.N || i == j) { ++bad; continue; }
        double r2 = 0.0;
#pragma unroll
        for (int c = 0; c < D; ++c) {
            const double d = __ldg(A.x + j * D + c) - __ldg(A.x + i * D + c);
            r2 = fma(d, d, r2);
        }
        const double e = sqrt(r2) - (A.r0 ? A.r0[s] : A.r0_u);
        u += 0.5 * (A.k ? A.k[s] : A.k_u) * e * e;
        ++live;
    }
    u = block_sum_d(u, shd);
    live = block_sum_u(live, shu);
    bad = block_sum_u(bad, shu);
    if (threadIdx.x == 0) {
        S.partU[blockIdx.x] = u;
        S.partN[blockIdx.x] = live;
        if (bad) atomicAdd(S.bad, bad);
    }
}

// Level 2: one block sums the nblk partials, thread t taking t, t + 1024, ... in that order, then the fixed-order block sum.
__global__ void __launch_bounds__(kSBlock) k_static_energy_final(unsigned char *scratch, int nblk, double *U, long long *counts) {
    __shared__ double shd[kSBlock / 32];
    __shared__ unsigned long long shu[kSBlock / 32];
    const StaticView S = view_of(scratch);
    double u = 0.0;
    unsigned long long live = 0;
    for (int c = threadIdx.x; c < nblk; c += kSBlock) { u += S.partU[c]; live += S.partN[c]; }
    u = block_sum_d(u, shd);
    live = block_sum_u(live, shu);
    if (threadIdx.x == 0) {
        *U = u;
        if (counts) { counts[0] = (long long)live; counts[1] = (long long)*S.bad; }
    }
}

// ---- host side -------------------------------------------------------------------------------------------------------
constexpr int kSMaxDevices = 64;
std::mutex g_setup_mutex;
unsigned char *g_scratch_addr[kSMaxDevices];      // device address of g_static_scratch on each device, looked up once
bool g_scratch_ready[kSMaxDevices];

lsm_status sfail(char *errbuf, size_t len, lsm_status st, const char *fmt, ...) {
    if (errbuf && len) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(errbuf, len, fmt, ap);
        va_end(ap);
    }
    return st;
}

struct StaticDeviceScope {   // makes `dev` current for the call, gives the caller's device back afterwards
    int prev = -1;
    cudaError_t err = cudaSuccess;
    explicit StaticDeviceScope(int dev) {
        err = cudaGetDevice(&prev);
        if (err != cudaSuccess) { prev = -1; return; }
        if (prev != dev) err = cudaSetDevice(dev); else prev = -1;
    }
    ~StaticDeviceScope() { if (prev >= 0) cudaSetDevice(prev); }
};

}  // namespace

extern "C" lsm_status lsm_spring_energy_static(int32_t device, void *stream, int32_t dim, int64_t n_particles, int64_t n_springs,
                                               const double *x, const int32_t *spring_i, const int32_t *spring_j,
                                               const double *k, const double *r0, double k_uniform, double r0_uniform,
                                               const uint8_t *broken, double *U, int64_t *counts, char *errbuf, size_t errbuf_len) {
    const char *me = "lsm_spring_energy_static";
    if (errbuf && errbuf_len) errbuf[0] = '\0';
    // argument checks first: none of them needs a CUDA device
    if (dim != 2 && dim != 3) return sfail(errbuf, errbuf_len, LSM_E_INVALID, "%s: dim must be 2 or 3 (got %d)", me, (int)dim);
    if (n_particles < 1 || n_particles >= 2147483647LL)
        return sfail(errbuf, errbuf_len, LSM_E_INVALID, "%s: n_particles must be in [1, 2^31 - 1) (got %lld)", me, (long long)n_particles);
    if (n_springs < 0) return sfail(errbuf, errbuf_len, LSM_E_INVALID, "%s: n_springs < 0", me);
    if (n_springs > (int64_t)LSM_STATIC_MAX_SPRINGS)
        return sfail(errbuf, errbuf_len, LSM_E_RANGE,
                     "%s: n_springs = %lld is above LSM_STATIC_MAX_SPRINGS = %lld, the most the library's fixed scratch array holds "
                     "partial sums for; nothing was computed (split the list and add the parts, or use lsm_create + lsm_read_energy)",
                     me, (long long)n_springs, (long long)LSM_STATIC_MAX_SPRINGS);
    if (!x || !U || (n_springs > 0 && (!spring_i || !spring_j)))
        return sfail(errbuf, errbuf_len, LSM_E_INVALID, "%s: x, U, spring_i and spring_j must not be NULL", me);
    if (device < 0 || device >= kSMaxDevices) return sfail(errbuf, errbuf_len, LSM_E_INVALID, "%s: device ordinal %d outside [0, %d)", me, (int)device, kSMaxDevices);

    StaticDeviceScope scope(device);
    if (scope.err != cudaSuccess)
        return sfail(errbuf, errbuf_len, LSM_E_CUDA, "%s: cannot make device %d current: %s (there is no CPU fallback)", me, (int)device, cudaGetErrorString(scope.err));

    // Set-up, once per device and with that device current: ask the runtime where THIS device keeps the array.
    unsigned char *scratch = nullptr;
    {
        std::lock_guard<std::mutex> lock(g_setup_mutex);
        if (!g_scratch_ready[device]) {
            void *p = nullptr;
            cudaError_t e = cudaGetSymbolAddress(&p, g_static_scratch);
            if (e != cudaSuccess || !p)
                return sfail(errbuf, errbuf_len, LSM_E_CUDA, "%s: cudaGetSymbolAddress(g_static_scratch) on device %d: %s", me, (int)device, cudaGetErrorString(e));
            g_scratch_addr[device] = static_cast<unsigned char *>(p);
            g_scratch_ready[device] = true;
        }
        scratch = g_scratch_addr[device];
    }

    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const int nblk = (int)((n_springs + kSChunk - 1) / kSChunk);
    cudaError_t e = cudaMemsetAsync(scratch, 0, sizeof(unsigned long long), st);       // the bad-id counter starts at zero
    if (e != cudaSuccess) return sfail(errbuf, errbuf_len, LSM_E_CUDA, "%s: cudaMemsetAsync: %s", me, cudaGetErrorString(e));
    if (nblk > 0) {
        EnergyArgs A;
        A.x = x; A.si = spring_i; A.sj = spring_j; A.k = k; A.r0 = r0; A.broken = broken;
        A.k_u = k_uniform; A.r0_u = r0_uniform; A.N = n_particles; A.M = n_springs;
        if (dim == 2) k_static_energy_partials<2><<<nblk, kSBlock, 0, st>>>(A, scratch);
        else k_static_energy_partials<3><<<nblk, kSBlock, 0, st>>>(A, scratch);
        e = cudaGetLastError();
        if (e != cudaSuccess) return sfail(errbuf, errbuf_len, LSM_E_CUDA, "%s: launch of the partial-sum kernel: %s", me, cudaGetErrorString(e));
    }
    k_static_energy_final<<<1, kSBlock, 0, st>>>(scratch, nblk, U, reinterpret_cast<long long *>(counts));
    e = cudaGetLastError();
    if (e != cudaSuccess) return sfail(errbuf, errbuf_len, LSM_E_CUDA, "%s: launch of the final-sum kernel: %s", me, cudaGetErrorString(e));
    return LSM_OK;
}
