// bench_peaks.cu -- roofline denominators for bench.py (libfdcpeaks.so).  MEASUREMENT TOOLING, not part of the
// method: nothing here is on the hot path and libfdc.so does not link it.  SURVEY §8(d) "Which roofline" asks for
// the measured rate of 64-bit reductions (`red.global.add.u64`, the deposit instruction of DESIGN.md R8;
// PAPER.md:L73 "blocked access to the memory location while a particular thread updated") from a saturating grid,
//   (i)   over uniformly random addresses in a buffer the size of a config's grid,
//   (ii)  with the lanes of a warp clustered on one sector / one word,
//   (iii) over a config's ACTUAL address multiset (a trace of the voxel indices the transport kernel sent its
//         reductions to, see fdc_trace_reds in include/fdc.h), replayed in trace order and in shuffled order.
// C-ABI, plain pointers and sizes; device pointers are said to be so.
#include <cuda_runtime.h>
#include <stdint.h>

namespace {

__device__ __forceinline__ uint64_t mix64(uint64_t x)
{ x ^= x >> 33; x *= 0xff51afd7ed558ccdULL; x ^= x >> 33; x *= 0xc4ceb9fe1a85ec53ULL; x ^= x >> 33; return x; }

// mode 0: uniform over n_words (a power of two); 1: the 32 lanes of a warp on 4 neighbouring words; 2: on one word
__global__ void k_peak_red(unsigned long long *buf, uint64_t n_words, uint64_t n_ops, int mode)
{
    const uint64_t tid = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x, nthr = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t op = tid; op < n_ops; op += nthr) {
        uint64_t a;
        if (mode == 0) a = mix64(op) & (n_words - 1);
        else if (mode == 1) a = ((mix64(op >> 5) & ((n_words >> 2) - 1)) << 2) + (op & 3);
        else a = mix64(op >> 5) & (n_words - 1);
        atomicAdd(buf + a, 1ull);
    }
}

// replay of a traced address list: every pass sends one reduction to each addr[i], i in grid-stride order.  The
// list is replayed as traced (consecutive entries were written by the lanes of one warp instruction, as the kernel
// issues them) or after k_permute has shuffled it (i -> (i * mult) mod n with mult coprime to n; untimed)
__global__ void k_replay_red(unsigned long long *buf, const uint32_t *__restrict__ addr, uint64_t n_addr, uint32_t passes)
{
    const uint64_t tid = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x, nthr = (uint64_t)gridDim.x * blockDim.x;
    for (uint32_t p = 0; p < passes; ++p)
        for (uint64_t i = tid; i < n_addr; i += nthr) atomicAdd(buf + addr[i], 1ull);
}
__global__ void k_permute(const uint32_t *__restrict__ in, uint32_t *__restrict__ out, uint64_t n, uint64_t mult)
{
    const uint64_t tid = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x, nthr = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t i = tid; i < n; i += nthr) out[i] = in[(uint64_t)(((unsigned __int128)i * mult) % n)];
}

uint64_t gcd64(uint64_t a, uint64_t b) { while (b) { const uint64_t t = a % b; a = b; b = t; } return a; }

int time_launch(int device, unsigned long long *buf, uint64_t bytes, double *ops_per_s, uint64_t n_ops,
                void (*launch)(int blocks, bool warm, void *), void *arg)
{
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return -5;
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    cudaMemset(buf, 0, bytes);
    const int blocks = prop.multiProcessorCount * 2;            // two resident blocks of 1024 threads per SM
    launch(blocks, true, arg);
    cudaEventRecord(e0);
    launch(blocks, false, arg);
    cudaEventRecord(e1);
    const cudaError_t e = cudaEventSynchronize(e1);
    float ms = 0.f; cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    if (e != cudaSuccess || cudaGetLastError() != cudaSuccess || !(ms > 0.f)) return -5;
    *ops_per_s = (double)n_ops / ((double)ms * 1e-3);
    return 0;
}

struct PeakArgs { unsigned long long *buf; uint64_t n_words, n_ops; int mode; };
struct ReplayArgs { unsigned long long *buf; const uint32_t *addr; uint64_t n_addr; uint32_t passes; };

}  // namespace

extern "C" {

// Uniform / clustered synthetic modes.  footprint_bytes is rounded down to a power of two.  Returns 0, -1 (bad
// argument), -4 (out of memory), -5 (CUDA error), -6 (not sm_100).
int fdcpeaks_red_u64(int device, uint64_t footprint_bytes, uint64_t n_ops, int mode, double *ops_per_s)
{
    if (!ops_per_s || footprint_bytes < 64 || n_ops == 0 || mode < 0 || mode > 2) return -1;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return -5;
    if (prop.major != 10) return -6;
    if (cudaSetDevice(device) != cudaSuccess) return -5;
    uint64_t n_words = 8;
    while (n_words * 2 * 8 <= footprint_bytes) n_words *= 2;
    unsigned long long *buf = nullptr;
    if (cudaMalloc(&buf, n_words * 8) != cudaSuccess) return -4;
    PeakArgs a{buf, n_words, n_ops, mode};
    const int rc = time_launch(device, buf, n_words * 8, ops_per_s, n_ops,
                               [](int blocks, bool warm, void *p) {
                                   const PeakArgs *a = static_cast<const PeakArgs *>(p);
                                   k_peak_red<<<blocks, 1024>>>(a->buf, a->n_words, warm ? a->n_ops / 8 + 1 : a->n_ops, a->mode);
                               }, &a);
    cudaFree(buf);
    return rc;
}

// Replay of a traced multiset.  addr_dev: DEVICE array of n_addr voxel indices, each < n_words (the library that
// wrote the trace guarantees it); the reductions go to a scratch buffer of n_words u64; the list is replayed
// `passes` times (operations = passes * n_addr).  shuffled = 0: trace order; 1: a fixed pseudo-random permutation.
int fdcpeaks_red_replay(int device, const uint32_t *addr_dev, uint64_t n_addr, uint64_t n_words, uint32_t passes, int shuffled,
                        double *ops_per_s)
{
    if (!ops_per_s || !addr_dev || n_addr == 0 || n_words == 0 || passes == 0) return -1;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return -5;
    if (prop.major != 10) return -6;
    if (cudaSetDevice(device) != cudaSuccess) return -5;
    unsigned long long *buf = nullptr;
    uint32_t *perm = nullptr;
    if (cudaMalloc(&buf, n_words * 8) != cudaSuccess) return -4;
    const uint32_t *src = addr_dev;
    if (shuffled) {                                              // about 0.618 n, made coprime to n
        uint64_t mult = (uint64_t)((double)n_addr * 0.6180339887498949) | 1ull;
        while (mult < n_addr && gcd64(mult, n_addr) != 1) mult += 2;
        if (mult >= n_addr) mult = 1;
        if (cudaMalloc(&perm, n_addr * 4) != cudaSuccess) { cudaFree(buf); return -4; }
        k_permute<<<prop.multiProcessorCount * 8, 256>>>(addr_dev, perm, n_addr, mult);
        src = perm;
    }
    ReplayArgs a{buf, src, n_addr, passes};
    const int rc = time_launch(device, buf, n_words * 8, ops_per_s, (uint64_t)passes * n_addr,
                               [](int blocks, bool warm, void *p) {
                                   const ReplayArgs *a = static_cast<const ReplayArgs *>(p);
                                   k_replay_red<<<blocks, 1024>>>(a->buf, a->addr, a->n_addr, warm ? 1u : a->passes);
                               }, &a);
    cudaFree(buf); cudaFree(perm);
    return rc;
}

}  // extern "C"
