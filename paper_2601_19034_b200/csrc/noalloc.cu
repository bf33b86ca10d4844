// noalloc.cu -- qnep_neutralise_noalloc (include/qnep.h): charge neutralisation, PAPER.md :255-262 Eq. 33 (DESIGN.md
// reading G3), for callers that must not allocate device memory.
//
// Who that is.  The rest of this library sizes its workspace with cudaMalloc (qnep_create, and again whenever the atom
// count or the mesh grows).  That is not an option for a caller that
//   - was handed a fixed slice of the GPU by its host application -- a plug-in of an MD engine or of an inference server
//     whose own pool allocator has already reserved the rest of the device, so that a raw cudaMalloc from a library either
//     fails or eats into memory the application counted on;
//   - runs in a section that must not stall the device: cudaMalloc and cudaFree may synchronise the whole context, which
//     serialises every other stream the application keeps busy;
//   - has to know its memory footprint before the first step and may not change it afterwards.
// For them the running sum that Eq. 33 needs lives in a small array that is part of the library image: it is reserved
// when the library is loaded on a GPU and given back when the process ends, and no call here ever allocates or frees.
//
// The existing path (k_nn* add sum_i q_i^raw into the handle's accumulator block, k_neutralise applies the shift;
// descriptor.cu) is untouched; this file shares no state with it.
#include <cuda_runtime.h>
#include <stdint.h>

#include <cstdio>
#include <mutex>

#include "../../include/qnep.h"

namespace {

constexpr int NOALLOC_THREADS = 256;
constexpr int NOALLOC_ATOMS_PER_BLOCK = 1024;                                          // four per thread
constexpr int NOALLOC_MAX_BLOCKS = QNEP_NOALLOC_MAX_ATOMS / NOALLOC_ATOMS_PER_BLOCK;   // 4096
static_assert(QNEP_NOALLOC_MAX_ATOMS % NOALLOC_ATOMS_PER_BLOCK == 0, "maximum must be a whole number of blocks");

// The scratch: one partial sum of q^raw per block of 1024 atoms, 4096 x 8 B = 32 KiB on every GPU that loads the
// library, until the process exits.  Every call on a device uses this one array, and it keeps whatever the last call
// left in it.  Nothing in it has to start at zero: a call writes slots 0 .. n_blocks-1 (k_noalloc_partial, every block
// unconditionally) before it reads exactly those slots (k_noalloc_apply), so leftovers of an earlier, larger call are
// never looked at and there is nothing to clear.  Two calls whose kernels overlap on the GPU (different streams without
// an event between them, or two host threads) overwrite each other's partial sums: the caller has to order them.
//
// In HOST code the name g_noalloc_partial is only a stand-in the runtime uses to look the array up; it is not a device
// address and must never be handed to a kernel.  The device address comes from cudaGetSymbolAddress (set-up below).
static __device__ __align__(256) double g_noalloc_partial[NOALLOC_MAX_BLOCKS];

__device__ __forceinline__ double block_total(double v, double* sh)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
    __syncthreads();
    double r = 0.0;
#pragma unroll
    for (int w = 0; w < NOALLOC_THREADS / 32; ++w) r += sh[w];        // same order in every thread of every block
    return r;
}

// partial[b] = sum of q^raw over atoms 1024 b .. 1024 b + 1023
__global__ void __launch_bounds__(NOALLOC_THREADS)
k_noalloc_partial(int64_t N, const double* __restrict__ qraw, double* __restrict__ partial)
{
    __shared__ double sh[NOALLOC_THREADS / 32];
    const int64_t base = (int64_t)blockIdx.x * NOALLOC_ATOMS_PER_BLOCK + threadIdx.x;
    double v = 0.0;
#pragma unroll
    for (int r = 0; r < NOALLOC_ATOMS_PER_BLOCK / NOALLOC_THREADS; ++r) {
        const int64_t i = base + (int64_t)r * NOALLOC_THREADS;
        if (i < N) v += qraw[i];
    }
    const double t = block_total(v, sh);
    if (threadIdx.x == 0) partial[blockIdx.x] = t;
}

// Eq. 33: q_i = q_i^raw + (Q - sum_j q_j^raw) / N.  Every block adds the n_blocks partial sums in the same order, so all
// atoms see the same shift to the last bit and the result does not depend on the launch.  out may alias qraw (each
// thread reads its atoms before it writes them).
__global__ void __launch_bounds__(NOALLOC_THREADS)
k_noalloc_apply(int64_t N, int n_blocks, const double* __restrict__ partial, double Qtot, const double* qraw, double* out)
{
    __shared__ double sh[NOALLOC_THREADS / 32];
    double v = 0.0;
    for (int k = threadIdx.x; k < n_blocks; k += NOALLOC_THREADS) v += partial[k];
    const double shift = (Qtot - block_total(v, sh)) / (double)N;
    const int64_t base = (int64_t)blockIdx.x * NOALLOC_ATOMS_PER_BLOCK + threadIdx.x;
#pragma unroll
    for (int r = 0; r < NOALLOC_ATOMS_PER_BLOCK / NOALLOC_THREADS; ++r) {
        const int64_t i = base + (int64_t)r * NOALLOC_THREADS;
        if (i < N) out[i] = qraw[i] + shift;
    }
}

// Set-up, once per device: the device address of the scratch array on THAT device (every device that loads the library
// has its own copy at its own address).
constexpr int NOALLOC_MAX_DEVICES = 64;
std::mutex g_setup_lock;
double* g_partial_addr[NOALLOC_MAX_DEVICES] = {nullptr};

void say(char* err, size_t len, const char* fmt, long long a = 0, long long b = 0)
{
    if (err && len) std::snprintf(err, len, fmt, a, b);
}

int scratch_of_current_device(double** out, char* err, size_t len)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { say(err, len, "qnep_neutralise_noalloc: cudaGetDevice failed (CUDA error %lld)", (long long)e); return QNEP_ERR_CUDA; }
    if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) { say(err, len, "qnep_neutralise_noalloc: device ordinal %lld is beyond the %lld this entry point keeps addresses for", dev, NOALLOC_MAX_DEVICES); return QNEP_ERR_UNSUPPORTED; }
    std::lock_guard<std::mutex> guard(g_setup_lock);
    if (!g_partial_addr[dev]) {
        double* p = nullptr;
        e = cudaGetSymbolAddress((void**)&p, g_noalloc_partial);          // with `dev` current: the copy on this device
        if (e != cudaSuccess || !p) {
            (void)cudaGetLastError();
            say(err, len, "qnep_neutralise_noalloc: cudaGetSymbolAddress failed on device %lld (CUDA error %lld)", dev, (long long)e);
            return QNEP_ERR_CUDA;
        }
        // load the two kernels now as well, so that later calls find everything in place
        cudaFuncAttributes fa;
        e = cudaFuncGetAttributes(&fa, k_noalloc_partial);
        if (e == cudaSuccess) e = cudaFuncGetAttributes(&fa, k_noalloc_apply);
        if (e != cudaSuccess) {
            (void)cudaGetLastError();
            say(err, len, "qnep_neutralise_noalloc: kernels not loadable on device %lld (CUDA error %lld)", dev, (long long)e);
            return QNEP_ERR_CUDA;
        }
        g_partial_addr[dev] = p;
    }
    *out = g_partial_addr[dev];
    return QNEP_OK;
}

}  // namespace

extern "C" int qnep_neutralise_noalloc(int64_t n_atoms, const double* q_raw_dev, double q_total, double* charges_dev,
                                       void* cuda_stream, char* err_host, size_t err_len)
{
    if (err_host && err_len) err_host[0] = '\0';
    if (!q_raw_dev || !charges_dev) { say(err_host, err_len, "qnep_neutralise_noalloc: null q_raw_dev or charges_dev"); return QNEP_ERR_INVALID_ARG; }
    if (n_atoms <= 0) { say(err_host, err_len, "qnep_neutralise_noalloc: n_atoms = %lld must be positive", (long long)n_atoms); return QNEP_ERR_INVALID_ARG; }
    if (n_atoms > (int64_t)QNEP_NOALLOC_MAX_ATOMS) {
        say(err_host, err_len, "qnep_neutralise_noalloc: n_atoms = %lld exceeds QNEP_NOALLOC_MAX_ATOMS = %lld, the size the built-in "
                               "scratch array was compiled for (use qnep_compute, which allocates, for larger systems)",
            (long long)n_atoms, (long long)QNEP_NOALLOC_MAX_ATOMS);
        return QNEP_ERR_UNSUPPORTED;
    }
    double* partial = nullptr;
    const int rc = scratch_of_current_device(&partial, err_host, err_len);
    if (rc != QNEP_OK) return rc;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const int nb = (int)((n_atoms + NOALLOC_ATOMS_PER_BLOCK - 1) / NOALLOC_ATOMS_PER_BLOCK);
    k_noalloc_partial<<<nb, NOALLOC_THREADS, 0, s>>>(n_atoms, q_raw_dev, partial);
    k_noalloc_apply<<<nb, NOALLOC_THREADS, 0, s>>>(n_atoms, nb, partial, q_total, q_raw_dev, charges_dev);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { say(err_host, err_len, "qnep_neutralise_noalloc: kernel launch failed (CUDA error %lld)", (long long)e); return QNEP_ERR_CUDA; }
    return QNEP_OK;
}
