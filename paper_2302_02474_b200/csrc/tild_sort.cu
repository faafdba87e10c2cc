// a1: canonical fp32 index map, cell keys, counting sort by cell, physical reorder.
// Not in the paper's PM text; nearest prior art is its neighbour-list cell binning with atomics
// (PAPER.md L205).  DESIGN.md A15/A16 define what is bit-exact.
#include "tild_internal.cuh"

namespace {

constexpr int SCAN_THREADS = 256;
constexpr int SCAN_ITEMS = 16;
constexpr int SCAN_CHUNK = SCAN_THREADS * SCAN_ITEMS;  // 4096 elements per block

template <int P>
__global__ void __launch_bounds__(256) cell_key_kernel(MeshParams m, const float* __restrict__ x,
                                                       uint32_t* __restrict__ key, int32_t* __restrict__ base)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= m.n) return;
    int c[3], b[3];
    float t;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        index_1d<P>(x[3 * (size_t)i + a], m.inv_h[a], c[a], b[a], t);
        c[a] = wrap_idx(c[a], m.N[a]);
    }
    if (key) key[i] = (uint32_t)((c[0] * m.N[1] + c[1]) * m.N[2] + c[2]);
    if (base) {
        base[3 * (size_t)i + 0] = b[0];
        base[3 * (size_t)i + 1] = b[1];
        base[3 * (size_t)i + 2] = b[2];
    }
}

// key = tile * TV + local cell (tile-major order; z fastest inside a tile so that consecutive particles share
// z-rows of the mesh, which is what the interpolation's loads want)
template <int P>
__global__ void __launch_bounds__(256) tile_key_kernel(MeshParams m, TileParams tp, const float* __restrict__ x,
                                                       const int32_t* __restrict__ type, uint32_t* __restrict__ key)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= m.n) return;
    int c[3], t[3], b;
    float off;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        index_1d<P>(x[3 * (size_t)i + a], m.inv_h[a], c[a], b, off);
        c[a] = wrap_idx(c[a], m.N[a]);
        t[a] = c[a] / tp.T[a];
        c[a] -= t[a] * tp.T[a];
    }
    const uint32_t tile = (uint32_t)((t[0] * tp.nt[1] + t[1]) * tp.nt[2] + t[2]);
    key[i] = (tile * (uint32_t)m.S + (uint32_t)type[i]) * (uint32_t)tp.TV + (uint32_t)((c[0] * tp.T[1] + c[1]) * tp.T[2] + c[2]);
}

__global__ void __launch_bounds__(256) gather_stage_kernel(int n, const uint32_t* __restrict__ perm,
                                                           const float* __restrict__ x0, const int32_t* __restrict__ t0,
                                                           float* __restrict__ x1, int32_t* __restrict__ t1)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n) return;
    const size_t o = perm[j];
    x1[3 * (size_t)j + 0] = x0[3 * o + 0];
    x1[3 * (size_t)j + 1] = x0[3 * o + 1];
    x1[3 * (size_t)j + 2] = x0[3 * o + 2];
    t1[j] = t0[o];
}

// count[key]++ ; rank[i] = arrival order inside the cell
__global__ void __launch_bounds__(256) histogram_kernel(int n, const uint32_t* __restrict__ key,
                                                        uint32_t* __restrict__ count, uint32_t* __restrict__ rank)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    rank[i] = atomicAdd(&count[key[i]], 1u);
}

__device__ __forceinline__ uint32_t warp_incl_scan(uint32_t v)
{
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const uint32_t o = __shfl_up_sync(0xffffffffu, v, d);
        if ((threadIdx.x & 31) >= d) v += o;
    }
    return v;
}

// exclusive scan of one value per thread across the block; returns the exclusive prefix, *total = block sum
template <int NT>
__device__ __forceinline__ uint32_t block_excl_scan(uint32_t v, uint32_t* total)
{
    __shared__ uint32_t warp_sums[NT / 32];
    __shared__ uint32_t block_total;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const uint32_t incl = warp_incl_scan(v);
    if (lane == 31) warp_sums[wid] = incl;
    __syncthreads();
    if (wid == 0) {
        uint32_t s = lane < NT / 32 ? warp_sums[lane] : 0u;
        const uint32_t si = warp_incl_scan(s);
        if (lane < NT / 32) warp_sums[lane] = si - s;
        if (lane == NT / 32 - 1) block_total = si;
    }
    __syncthreads();
    const uint32_t r = warp_sums[wid] + incl - v;
    if (total) *total = block_total;
    __syncthreads();
    return r;
}

__global__ void __launch_bounds__(SCAN_THREADS) scan_reduce_kernel(size_t len, const uint32_t* __restrict__ in,
                                                                   uint32_t* __restrict__ part)
{
    const size_t start = (size_t)blockIdx.x * SCAN_CHUNK;
    uint32_t s = 0;
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        const size_t j = start + (size_t)k * SCAN_THREADS + threadIdx.x;
        if (j < len) s += in[j];
    }
    uint32_t total;
    block_excl_scan<SCAN_THREADS>(s, &total);
    if (threadIdx.x == 0) part[blockIdx.x] = total;
}

// single block: exclusive scan of part[0..nb) in place
__global__ void __launch_bounds__(1024) scan_parts_kernel(int nb, uint32_t* __restrict__ part)
{
    const int per = (nb + 1023) / 1024;
    const int lo = threadIdx.x * per;
    uint32_t s = 0;
    for (int k = 0; k < per; ++k)
        if (lo + k < nb) s += part[lo + k];
    uint32_t run = block_excl_scan<1024>(s, nullptr);
    for (int k = 0; k < per; ++k)
        if (lo + k < nb) {
            const uint32_t v = part[lo + k];
            part[lo + k] = run;
            run += v;
        }
}

__global__ void __launch_bounds__(SCAN_THREADS) scan_final_kernel(size_t len, const uint32_t* __restrict__ in,
                                                                  const uint32_t* __restrict__ part,
                                                                  uint32_t* __restrict__ out)
{
    const size_t start = (size_t)blockIdx.x * SCAN_CHUNK + (size_t)threadIdx.x * SCAN_ITEMS;
    uint32_t v[SCAN_ITEMS];
    uint32_t s = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        v[k] = start + k < len ? in[start + k] : 0u;
        s += v[k];
    }
    uint32_t run = block_excl_scan<SCAN_THREADS>(s, nullptr) + part[blockIdx.x];
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        if (start + k < len) out[start + k] = run;
        run += v[k];
    }
}

// perm[cell_start[key] + rank] = i ; rank[i] <- destination (the inverse permutation)
__global__ void __launch_bounds__(256) scatter_kernel(int n, const uint32_t* __restrict__ key,
                                                      const uint32_t* __restrict__ cell_start,
                                                      uint32_t* __restrict__ rank, uint32_t* __restrict__ perm)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const uint32_t dst = cell_start[key[i]] + rank[i];
    perm[dst] = (uint32_t)i;
    rank[i] = dst;
}

// new particle j = old particle perm[j]; bond partners remapped through inv = rank
__global__ void __launch_bounds__(256) reorder_kernel(int n, int max_bonds, const uint32_t* __restrict__ perm,
                                                      const uint32_t* __restrict__ inv, const float* __restrict__ x0,
                                                      const float* __restrict__ w0, const int32_t* __restrict__ t0,
                                                      const uint32_t* __restrict__ id0, const int32_t* __restrict__ b0,
                                                      float* __restrict__ x1, float* __restrict__ w1,
                                                      int32_t* __restrict__ t1, uint32_t* __restrict__ id1,
                                                      int32_t* __restrict__ b1)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n) return;
    const size_t o = perm[j];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        x1[3 * (size_t)j + a] = x0[3 * o + a];
        w1[3 * (size_t)j + a] = w0[3 * o + a];
    }
    t1[j] = t0[o];
    id1[j] = id0[o];
    for (int s = 0; s < max_bonds; ++s) {
        const int32_t q = b0[o * max_bonds + s];
        b1[(size_t)j * max_bonds + s] = q < 0 ? -1 : (int32_t)inv[q];
    }
}

// dst[id[i]][:] = src[i][:]
__global__ void __launch_bounds__(256) unpermute_kernel(int n, int ncomp, const uint32_t* __restrict__ id,
                                                        const float* __restrict__ src, float* __restrict__ dst)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const size_t o = id[i];
    for (int a = 0; a < ncomp; ++a) dst[o * ncomp + a] = src[(size_t)i * ncomp + a];
}

}  // namespace

int launch_cell_keys(tild_ctx* c, const float* x, uint32_t* key, int32_t* base)
{
    const int n = c->mesh.n;
    if (n == 0) return TILD_OK;
    const int nb = (n + 255) / 256;
    switch (c->mesh.P) {
    case 1: cell_key_kernel<1><<<nb, 256, 0, c->stream>>>(c->mesh, x, key, base); break;
    case 2: cell_key_kernel<2><<<nb, 256, 0, c->stream>>>(c->mesh, x, key, base); break;
    case 3: cell_key_kernel<3><<<nb, 256, 0, c->stream>>>(c->mesh, x, key, base); break;
    default: cell_key_kernel<4><<<nb, 256, 0, c->stream>>>(c->mesh, x, key, base); break;
    }
    TILD_LAUNCH_CHECK(c, "cell_key_kernel");
    return TILD_OK;
}

// Counting sort by cell key: histogram (arrival rank per particle) -> exclusive scan -> scatter.
// Scratch: count = c->cell_fill [M+1]; c->scan_part holds the nbs block sums followed by rank[n]; after the
// scatter rank[i] is the destination of particle i, i.e. the inverse permutation used by launch_reorder.
int launch_tile_keys(tild_ctx* c, const float* x, const int32_t* type, uint32_t* key)
{
    const int n = c->mesh.n;
    if (n == 0) return TILD_OK;
    const int nb = (n + 255) / 256;
    switch (c->mesh.P) {
    case 1: tile_key_kernel<1><<<nb, 256, 0, c->stream>>>(c->mesh, c->tile, x, type, key); break;
    case 2: tile_key_kernel<2><<<nb, 256, 0, c->stream>>>(c->mesh, c->tile, x, type, key); break;
    case 3: tile_key_kernel<3><<<nb, 256, 0, c->stream>>>(c->mesh, c->tile, x, type, key); break;
    default: tile_key_kernel<4><<<nb, 256, 0, c->stream>>>(c->mesh, c->tile, x, type, key); break;
    }
    TILD_LAUNCH_CHECK(c, "tile_key_kernel");
    return TILD_OK;
}

int launch_counting_sort(tild_ctx* c, const uint32_t* key, size_t nbins, uint32_t* perm, uint32_t* start)
{
    const int n = c->mesh.n;
    const size_t len = nbins + 1;
    const int nbs = (int)((len + SCAN_CHUNK - 1) / SCAN_CHUNK);
    uint32_t* count = c->cell_fill;
    uint32_t* part = c->scan_part;
    uint32_t* rank = c->scan_part + (c->max_bins + 1 + SCAN_CHUNK - 1) / SCAN_CHUNK;  // fixed offset: see launch_reorder
    TILD_CUDA(c, cudaMemsetAsync(count, 0, len * sizeof(uint32_t), c->stream));
    if (n > 0) {
        histogram_kernel<<<(n + 255) / 256, 256, 0, c->stream>>>(n, key, count, rank);
        TILD_LAUNCH_CHECK(c, "histogram_kernel");
    }
    scan_reduce_kernel<<<nbs, SCAN_THREADS, 0, c->stream>>>(len, count, part);
    TILD_LAUNCH_CHECK(c, "scan_reduce_kernel");
    scan_parts_kernel<<<1, 1024, 0, c->stream>>>(nbs, part);
    TILD_LAUNCH_CHECK(c, "scan_parts_kernel");
    scan_final_kernel<<<nbs, SCAN_THREADS, 0, c->stream>>>(len, count, part, start);
    TILD_LAUNCH_CHECK(c, "scan_final_kernel");
    if (n > 0 && perm) {
        scatter_kernel<<<(n + 255) / 256, 256, 0, c->stream>>>(n, key, start, rank, perm);
        TILD_LAUNCH_CHECK(c, "scatter_kernel");
    }
    return TILD_OK;
}

int launch_reorder(tild_ctx* c)
{
    const int n = c->mesh.n;
    int rc = launch_tile_keys(c, c->x[c->cur], c->type[c->cur], c->key);
    if (rc) return rc;
    rc = launch_counting_sort(c, c->key, c->tile.nbins, c->perm, c->tile_start);
    if (rc) return rc;
    c->steps_since_sort = 0;
    if (n == 0) return TILD_OK;
    const uint32_t* inv = c->scan_part + (c->max_bins + 1 + SCAN_CHUNK - 1) / SCAN_CHUNK;
    const int a = c->cur, b = 1 - c->cur;
    reorder_kernel<<<(n + 255) / 256, 256, 0, c->stream>>>(n, c->stp.max_bonds, c->perm, inv, c->x[a], c->w[a], c->type[a],
                                                           c->id[a], c->bond[a], c->x[b], c->w[b], c->type[b], c->id[b],
                                                           c->bond[b]);
    TILD_LAUNCH_CHECK(c, "reorder_kernel");
    c->cur = b;
    return TILD_OK;
}

int launch_stage_sort(tild_ctx* c, const float* x, const int32_t* type)
{
    const int n = c->mesh.n;
    int rc = launch_tile_keys(c, x, type, c->key);
    if (rc) return rc;
    rc = launch_counting_sort(c, c->key, c->tile.nbins, c->perm, c->cell_start);
    if (rc || n == 0) return rc;
    gather_stage_kernel<<<(n + 255) / 256, 256, 0, c->stream>>>(n, c->perm, x, type, c->stage_x, c->stage_type);
    TILD_LAUNCH_CHECK(c, "gather_stage_kernel");
    return TILD_OK;
}

int launch_unpermute(tild_ctx* c, const float* src, float* dst, int ncomp)
{
    const int n = c->mesh.n;
    if (n == 0) return TILD_OK;
    unpermute_kernel<<<(n + 255) / 256, 256, 0, c->stream>>>(n, ncomp, c->id[c->cur], src, dst);
    TILD_LAUNCH_CHECK(c, "unpermute_kernel");
    return TILD_OK;
}

size_t tild_scan_scratch_entries(size_t nbins, int n)
{
    const size_t len = nbins + 1;
    return (len + SCAN_CHUNK - 1) / SCAN_CHUNK + (size_t)n + 16;
}
