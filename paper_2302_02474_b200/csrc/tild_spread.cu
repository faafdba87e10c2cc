// a2: particle -> mesh spread.  PAPER.md L223: "at each time-step, every particle assigns
// its density contribution to nearby grid points, using a spline interpolation scheme"; Eq. 1 L110.
// grid[J][g] = sum_{i in J} W_x W_y W_z  (raw weights), g = (ix*Ny + iy)*Nz + iz.
//
// Hot kernel: one CTA per tile of TX x TY x TZ cells.  Particles are kept physically sorted by tile
// (tild_sort.cu), so the CTA's particles are one contiguous range.  The P^3 stencil of every particle is
// accumulated into a shared-memory tile (tile + stencil halo + drift margin) and the tile is flushed to the
// global grid once, so global-atomic traffic is per tile node instead of per particle.
//
// sm_100a has no native fp32 shared-memory atomic add (atomicAdd(float*) on shared compiles to an
// LDS + FADD + ATOMS.CAST.SPIN loop) but does have a native 32-bit integer one (ATOMS.ADD).  The tile is
// therefore accumulated in unsigned 2^-24 fixed point: each contribution is rounded once to 2^-24 (finer than
// an fp32 running sum near 1), the integer sum is exact and order-independent, and it is converted to fp32 at
// the flush.  A tile node holds < 256; a wrap is detected exactly by the tile's mass balance
// (sum of the tile == particles * 2^24 up to rounding) and such a tile is redone with fp32 global atomics.
// Measured on B200 (profiles/): fp32 CAS tile 1.09 ms, u32 tile 0.37-0.50 ms, per-particle global 1.34 ms (C4).
#include "tild_internal.cuh"

namespace {

constexpr int SPREAD_THREADS = 256;
constexpr float FIX_SCALE = 16777216.0f;       // 2^24
constexpr float FIX_INV = 1.0f / 16777216.0f;

// Baseline / fallback: one thread per particle, P^3 global reductions (REDG.E.ADD.F32 resolves in L2).
template <int P>
__device__ __forceinline__ void spread_global_one(const MeshParams& m, const int b[3], const float w[3][P], float* __restrict__ g,
                                                  float sign)
{
    int iz[P];
#pragma unroll
    for (int j = 0; j < P; ++j) iz[j] = wrap_idx(b[2] + j, m.N[2]);
#pragma unroll
    for (int jx = 0; jx < P; ++jx) {
        const size_t ox = (size_t)wrap_idx(b[0] + jx, m.N[0]) * m.N[1];
#pragma unroll
        for (int jy = 0; jy < P; ++jy) {
            const size_t row = (ox + wrap_idx(b[1] + jy, m.N[1])) * m.N[2];
            const float wxy = sign * w[0][jx] * w[1][jy];
#pragma unroll
            for (int jz = 0; jz < P; ++jz) atomicAdd(g + row + iz[jz], wxy * w[2][jz]);
        }
    }
}

template <int P>
__global__ void __launch_bounds__(256) spread_naive_kernel(MeshParams m, const float* __restrict__ x,
                                                           const int32_t* __restrict__ type, float* __restrict__ grid)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= m.n) return;
    int cell, b[3];
    float t, w[3][P];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        index_1d<P>(x[3 * (size_t)i + a], m.inv_h[a], cell, b[a], t);
        weights_1d<P>(t, w[a]);
    }
    spread_global_one<P>(m, b, w, grid + (size_t)type[i] * m.M, 1.0f);
}

__device__ __forceinline__ unsigned long long block_sum_u64(unsigned long long v, unsigned long long* scratch)
{
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    __syncthreads();
    if (lane == 0) scratch[wid] = v;
    __syncthreads();
    unsigned long long s = 0;
    for (int k = 0; k < SPREAD_THREADS / 32; ++k) s += scratch[k];
    return s;
}

template <int P>
__global__ void __launch_bounds__(SPREAD_THREADS) spread_tile_kernel(MeshParams m, TileParams tp,
                                                                     const uint32_t* __restrict__ cell_start,
                                                                     const float* __restrict__ x,
                                                                     const int32_t* __restrict__ type,
                                                                     float* __restrict__ grid)
{
    extern __shared__ uint32_t sm[];
    __shared__ unsigned long long red[SPREAD_THREADS / 32];
    const int EX = tp.E[0], EY = tp.E[1], EZ = tp.E[2];
    const int E3 = EX * EY * EZ;
    const int tile = blockIdx.x;
    const int tz = tile % tp.nt[2], ty = (tile / tp.nt[2]) % tp.nt[1], tx = tile / (tp.nt[2] * tp.nt[1]);
    const int o[3] = {tx * tp.T[0] - tp.lo, ty * tp.T[1] - tp.lo, tz * tp.T[2] - tp.lo};
    const uint32_t p_lo = cell_start[(size_t)tile * tp.TV], p_hi = cell_start[(size_t)(tile + 1) * tp.TV];
    if (p_lo == p_hi) return;

    for (int k = threadIdx.x; k < m.S * E3; k += SPREAD_THREADS) sm[k] = 0u;
    __syncthreads();

    uint32_t n_tile = 0;  // particles this thread accumulated through shared memory
    for (uint32_t i = p_lo + threadIdx.x; i < p_hi; i += SPREAD_THREADS) {
        int cell, b[3], d[3];
        float t, w[3][P];
        bool inside = true;
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            index_1d<P>(x[3 * (size_t)i + a], m.inv_h[a], cell, b[a], t);
            weights_1d<P>(t, w[a]);
            d[a] = wrap_idx(b[a] - o[a], m.N[a]);   // local node of the stencil's first node (any periodic image)
            inside = inside && (d[a] + P <= tp.E[a]);
        }
        const int ty_i = type[i];
        if (inside) {
            uint32_t* s = sm + ty_i * E3 + (d[0] * EY + d[1]) * EZ + d[2];
#pragma unroll
            for (int jx = 0; jx < P; ++jx)
#pragma unroll
                for (int jy = 0; jy < P; ++jy) {
                    const float wxy = w[0][jx] * w[1][jy] * FIX_SCALE;
#pragma unroll
                    for (int jz = 0; jz < P; ++jz) atomicAdd(s + (jx * EY + jy) * EZ + jz, __float2uint_rn(wxy * w[2][jz]));
                }
            ++n_tile;
        } else {
            // drifted out of the tile's halo since the last re-sort: rare, goes straight to the global grid
            spread_global_one<P>(m, b, w, grid + (size_t)ty_i * m.M, 1.0f);
        }
    }
    __syncthreads();

    // flush: one warp per z-row of the tile so that the global reductions are coalesced along z
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int rows = m.S * EX * EY;
    unsigned long long tile_sum = 0;
    for (int pass = 0; pass < 2; ++pass) {          // pass 1 only runs to undo a wrapped tile
        const float sc = pass == 0 ? FIX_INV : -FIX_INV;
        for (int r = wid; r < rows; r += SPREAD_THREADS / 32) {
            const int s = r / (EX * EY), q = r - s * (EX * EY);
            const int lx = q / EY, ly = q - lx * EY;
            float* grow = grid + (size_t)s * m.M +
                          ((size_t)wrap_idx(o[0] + lx, m.N[0]) * m.N[1] + wrap_idx(o[1] + ly, m.N[1])) * m.N[2];
            const uint32_t* srow = sm + (size_t)r * EZ;
            for (int lz = lane; lz < EZ; lz += 32) {
                const uint32_t u = srow[lz];
                if (u) {
                    if (pass == 0) tile_sum += u;
                    atomicAdd(grow + wrap_idx(o[2] + lz, m.N[2]), (float)u * sc);
                }
            }
        }
        if (pass == 1) break;
        const unsigned long long total = block_sum_u64(tile_sum, red);
        const unsigned long long cnt = block_sum_u64((unsigned long long)n_tile, red);
        const unsigned long long expect = cnt << 24, slack = 64ull * cnt + 64ull;
        const bool ok = total + slack >= expect && total <= expect + slack;
        if (ok) return;                               // uniform across the block
    }
    // a node wrapped past 2^32 (>= 256 particles' worth on one node): redo this tile with fp32 global atomics
    for (uint32_t i = p_lo + threadIdx.x; i < p_hi; i += SPREAD_THREADS) {
        int cell, b[3];
        float t, w[3][P];
        bool inside = true;
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            index_1d<P>(x[3 * (size_t)i + a], m.inv_h[a], cell, b[a], t);
            weights_1d<P>(t, w[a]);
            inside = inside && (wrap_idx(b[a] - o[a], m.N[a]) + P <= tp.E[a]);
        }
        if (inside) spread_global_one<P>(m, b, w, grid + (size_t)type[i] * m.M, 1.0f);
    }
}

}  // namespace

int launch_spread_naive(tild_ctx* c, const float* x, const int32_t* type, float* grid)
{
    const int n = c->mesh.n;
    TILD_CUDA(c, cudaMemsetAsync(grid, 0, sizeof(float) * c->M * c->mesh.S, c->stream));
    if (n == 0) return TILD_OK;
    const int nb = (n + 255) / 256;
    switch (c->mesh.P) {
    case 1: spread_naive_kernel<1><<<nb, 256, 0, c->stream>>>(c->mesh, x, type, grid); break;
    case 2: spread_naive_kernel<2><<<nb, 256, 0, c->stream>>>(c->mesh, x, type, grid); break;
    case 3: spread_naive_kernel<3><<<nb, 256, 0, c->stream>>>(c->mesh, x, type, grid); break;
    default: spread_naive_kernel<4><<<nb, 256, 0, c->stream>>>(c->mesh, x, type, grid); break;
    }
    TILD_LAUNCH_CHECK(c, "spread_naive_kernel");
    return TILD_OK;
}

int tild_spread_configure(tild_ctx* c)
{
    const size_t bytes = c->tile.smem_bytes;
    cudaError_t e = cudaSuccess;
    if (e == cudaSuccess) e = cudaFuncSetAttribute(spread_tile_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(spread_tile_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(spread_tile_kernel<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(spread_tile_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    if (e != cudaSuccess) return tild_fail(c, TILD_ECUDA, "cudaFuncSetAttribute(spread_tile_kernel, %zu B): %s", bytes, cudaGetErrorString(e));
    return TILD_OK;
}

// x/type must be sorted by tile with cell_start = the tile-major counting-sort offsets (launch_tile_sort).
int launch_spread_tiled(tild_ctx* c, const uint32_t* cell_start, const float* x, const int32_t* type, float* grid)
{
    TILD_CUDA(c, cudaMemsetAsync(grid, 0, sizeof(float) * c->M * c->mesh.S, c->stream));
    if (c->mesh.n == 0) return TILD_OK;
    const TileParams& tp = c->tile;
    const size_t sm = tp.smem_bytes;
    switch (c->mesh.P) {
    case 1: spread_tile_kernel<1><<<tp.ntiles, SPREAD_THREADS, sm, c->stream>>>(c->mesh, tp, cell_start, x, type, grid); break;
    case 2: spread_tile_kernel<2><<<tp.ntiles, SPREAD_THREADS, sm, c->stream>>>(c->mesh, tp, cell_start, x, type, grid); break;
    case 3: spread_tile_kernel<3><<<tp.ntiles, SPREAD_THREADS, sm, c->stream>>>(c->mesh, tp, cell_start, x, type, grid); break;
    default: spread_tile_kernel<4><<<tp.ntiles, SPREAD_THREADS, sm, c->stream>>>(c->mesh, tp, cell_start, x, type, grid); break;
    }
    TILD_LAUNCH_CHECK(c, "spread_tile_kernel");
    return TILD_OK;
}
