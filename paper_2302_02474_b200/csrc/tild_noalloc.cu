// tild_cell_start_noalloc (include/tild.h): the cell offsets of the a1 index map -- histogram of the cell keys + exclusive
// scan, the first half of the counting sort of tild_sort.cu -- for callers that cannot allocate: code under CUDA graph
// capture, serving loops, harnesses that forbid cudaMalloc.  No context, no workspace: the scan's block partials, which
// the context path keeps in the caller's workspace (tild_ctx::scan_part), live in a file-scope __device__ array of a
// fixed maximum size that every GPU loading the library holds until exit.
//
// The entry point calls no cudaMalloc / cudaFree and no allocating library routine (it runs one memset and four kernels on
// the caller's stream).  Every call shares the one array: it is fully rewritten before it is read (nothing in it has to
// start at zero, nothing is kept between calls), and two calls that overlap on the GPU (different streams, no ordering
// between them) race on it.
#include <cuda_runtime.h>

#include <mutex>
#include <stdarg.h>
#include <stdint.h>
#include <stdio.h>

#include "../../include/tild.h"

namespace {

constexpr int NA_THREADS = 256;                       // threads per scan block
constexpr int NA_ITEMS = 16;                          // entries per thread
constexpr int NA_CHUNK = NA_THREADS * NA_ITEMS;       // entries per scan block
constexpr int NA_MAX_PARTS = 4097;                    // blocks for TILD_NOALLOC_MAX_CELLS + 1 entries
static_assert((size_t)NA_MAX_PARTS * NA_CHUNK >= (size_t)TILD_NOALLOC_MAX_CELLS + 1, "partials cover the maximum size");

// 16.4 KB per GPU.  In host code this name is a host-side stand-in, not a device address: the launches below get the
// address cudaGetSymbolAddress returns for the current device (scratch_for_current_device).
static __device__ __align__(256) uint32_t na_scan_part[NA_MAX_PARTS];

constexpr int NA_MAX_DEVICES = 64;
std::mutex na_mu;
uint32_t* na_part_of_device[NA_MAX_DEVICES];          // device address of na_scan_part per device, looked up once

// count[key]++ for keys inside [0, n_cells); the others are counted in *n_bad (when given) and left out
__global__ void __launch_bounds__(256) na_histogram_kernel(int n, uint32_t n_cells, const uint32_t* __restrict__ key,
                                                           uint32_t* __restrict__ count, uint32_t* __restrict__ n_bad)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const uint32_t k = key[i];
    if (k < n_cells) atomicAdd(&count[k], 1u);
    else if (n_bad) atomicAdd(n_bad, 1u);
}

__device__ __forceinline__ uint32_t na_warp_incl_scan(uint32_t v)
{
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const uint32_t o = __shfl_up_sync(0xffffffffu, v, d);
        if ((threadIdx.x & 31) >= d) v += o;
    }
    return v;
}

// exclusive prefix of one value per thread across the block; *total (thread 0's copy is what callers use) = block sum
template <int NT>
__device__ __forceinline__ uint32_t na_block_excl_scan(uint32_t v, uint32_t* total)
{
    __shared__ uint32_t warp_sums[NT / 32];
    __shared__ uint32_t block_total;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const uint32_t incl = na_warp_incl_scan(v);
    if (lane == 31) warp_sums[wid] = incl;
    __syncthreads();
    if (wid == 0) {
        const uint32_t s = lane < NT / 32 ? warp_sums[lane] : 0u;
        const uint32_t si = na_warp_incl_scan(s);
        if (lane < NT / 32) warp_sums[lane] = si - s;
        if (lane == NT / 32 - 1) block_total = si;
    }
    __syncthreads();
    const uint32_t r = warp_sums[wid] + incl - v;
    if (total) *total = block_total;
    __syncthreads();
    return r;
}

// part[b] = sum of block b's NA_CHUNK entries
__global__ void __launch_bounds__(NA_THREADS) na_scan_reduce_kernel(size_t len, const uint32_t* __restrict__ in, uint32_t* __restrict__ part)
{
    const size_t start = (size_t)blockIdx.x * NA_CHUNK;
    uint32_t s = 0;
    for (int k = 0; k < NA_ITEMS; ++k) {
        const size_t j = start + (size_t)k * NA_THREADS + threadIdx.x;
        if (j < len) s += in[j];
    }
    uint32_t total;
    na_block_excl_scan<NA_THREADS>(s, &total);
    if (threadIdx.x == 0) part[blockIdx.x] = total;
}

// one block: exclusive scan of part[0..nb) in place
__global__ void __launch_bounds__(1024) na_scan_parts_kernel(int nb, uint32_t* __restrict__ part)
{
    const int per = (nb + 1023) / 1024;
    const int lo = threadIdx.x * per;
    uint32_t s = 0;
    for (int k = 0; k < per; ++k)
        if (lo + k < nb) s += part[lo + k];
    uint32_t run = na_block_excl_scan<1024>(s, nullptr);
    for (int k = 0; k < per; ++k)
        if (lo + k < nb) {
            const uint32_t v = part[lo + k];
            part[lo + k] = run;
            run += v;
        }
}

// data[j] <- number of entries before j, in place (a thread reads its NA_ITEMS consecutive entries before it writes them)
__global__ void __launch_bounds__(NA_THREADS) na_scan_final_kernel(size_t len, uint32_t* __restrict__ data, const uint32_t* __restrict__ part)
{
    const size_t start = (size_t)blockIdx.x * NA_CHUNK + (size_t)threadIdx.x * NA_ITEMS;
    uint32_t v[NA_ITEMS];
    uint32_t s = 0;
#pragma unroll
    for (int k = 0; k < NA_ITEMS; ++k) {
        v[k] = start + k < len ? data[start + k] : 0u;
        s += v[k];
    }
    uint32_t run = na_block_excl_scan<NA_THREADS>(s, nullptr) + part[blockIdx.x];
#pragma unroll
    for (int k = 0; k < NA_ITEMS; ++k) {
        if (start + k < len) data[start + k] = run;
        run += v[k];
    }
}

int na_fail(char* errmsg, size_t errmsg_len, int code, const char* fmt, ...)
{
    if (errmsg && errmsg_len > 0) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(errmsg, errmsg_len, fmt, ap);
        va_end(ap);
    }
    return code;
}

// device address of the scratch array on the CURRENT device; looked up once per device
cudaError_t scratch_for_current_device(uint32_t** out, int* device)
{
    cudaError_t e = cudaGetDevice(device);
    if (e != cudaSuccess) return e;
    if (*device < 0 || *device >= NA_MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lk(na_mu);
    if (!na_part_of_device[*device]) {
        uint32_t* p = nullptr;
        e = cudaGetSymbolAddress(reinterpret_cast<void**>(&p), na_scan_part);
        if (e != cudaSuccess) return e;
        na_part_of_device[*device] = p;
    }
    *out = na_part_of_device[*device];
    return cudaSuccess;
}

}  // namespace

extern "C" int tild_cell_start_noalloc(const uint32_t* cell_key, int32_t n, uint32_t n_cells, uint32_t* cell_start, uint32_t* n_bad,
                                       void* stream, char* errmsg, size_t errmsg_len)
{
    if (errmsg && errmsg_len > 0) errmsg[0] = '\0';
    if (n < 0 || n_cells == 0 || !cell_start || (n > 0 && !cell_key))
        return na_fail(errmsg, errmsg_len, TILD_EINVAL, "tild_cell_start_noalloc: n < 0, n_cells == 0 or a null argument");
    if (n_cells > (uint32_t)TILD_NOALLOC_MAX_CELLS)
        return na_fail(errmsg, errmsg_len, TILD_EINVAL,
                       "tild_cell_start_noalloc: n_cells = %u exceeds TILD_NOALLOC_MAX_CELLS = %d (the static scratch array holds the "
                       "scan partials of at most that many cells); use tild_index_map with a context",
                       n_cells, TILD_NOALLOC_MAX_CELLS);
    uint32_t* part = nullptr;
    int device = -1;
    cudaError_t e = scratch_for_current_device(&part, &device);
    if (e != cudaSuccess)
        return na_fail(errmsg, errmsg_len, TILD_ECUDA, "tild_cell_start_noalloc: cudaGetSymbolAddress on device %d: %s", device, cudaGetErrorString(e));
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const size_t len = (size_t)n_cells + 1;
    const int nbs = (int)((len + NA_CHUNK - 1) / NA_CHUNK);
    // the counts are accumulated in the caller's output array and scanned in place; the only scratch is the block partials
    e = cudaMemsetAsync(cell_start, 0, len * sizeof(uint32_t), st);
    if (e == cudaSuccess && n_bad) e = cudaMemsetAsync(n_bad, 0, sizeof(uint32_t), st);
    if (e != cudaSuccess) return na_fail(errmsg, errmsg_len, TILD_ECUDA, "tild_cell_start_noalloc: cudaMemsetAsync: %s", cudaGetErrorString(e));
    if (n > 0) na_histogram_kernel<<<(n + 255) / 256, 256, 0, st>>>(n, n_cells, cell_key, cell_start, n_bad);
    na_scan_reduce_kernel<<<nbs, NA_THREADS, 0, st>>>(len, cell_start, part);
    na_scan_parts_kernel<<<1, 1024, 0, st>>>(nbs, part);
    na_scan_final_kernel<<<nbs, NA_THREADS, 0, st>>>(len, cell_start, part);
    e = cudaGetLastError();
    if (e != cudaSuccess) return na_fail(errmsg, errmsg_len, TILD_ECUDA, "tild_cell_start_noalloc: kernel launch: %s", cudaGetErrorString(e));
    return TILD_OK;
}
