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
// therefore accumulated in unsigned 2^-23 fixed point: each contribution is rounded once to 2^-23 (read off the
// mantissa of 1 + w, so no F2I on the XU pipe), the integer sum is exact and order-independent, and it is
// converted to fp32 at the flush.  A tile node holds < 512; a wrap is detected exactly by the tile's mass balance
// (sum of the tile == particles * 2^23 up to rounding) and such a tile is redone with fp32 global atomics.
// Measured on B200 (profiles/): fp32 CAS tile 1.09 ms, u32 tile 0.37-0.50 ms, per-particle global 1.34 ms (C4).
#include "tild_internal.cuh"

namespace {

constexpr int SPREAD_THREADS = 256;
constexpr int FIX_BITS = 23;                    // tile fixed point: units of 2^-23
constexpr float FIX_INV = 1.0f / 8388608.0f;

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

// Tile edge in x and y is fixed at 8 cells; EZ = TZ + halo is a template parameter so that every shared-memory
// offset of the stencil is an immediate (the runtime-stride version spent 3/4 of its instructions on addresses).
template <int P, int EZ>
__global__ void __launch_bounds__(SPREAD_THREADS) spread_tile_kernel(MeshParams m, TileParams tp,
                                                                     const uint32_t* __restrict__ cell_start,
                                                                     const float* __restrict__ x, float* __restrict__ grid)
{
    constexpr int HALO = (P >= 3) ? 3 : 1;
    constexpr int EX = 8 + HALO, EY = 8 + HALO;
    constexpr int E3 = EX * EY * EZ;
    extern __shared__ __align__(16) uint32_t sm[];
    __shared__ unsigned long long red[SPREAD_THREADS / 32];
    __shared__ int goff_x[EX], goff_y[EY];         // wrapped global x / y node of each local x / y
    const int tile = blockIdx.x;
    const int tz = tile % tp.nt[2], ty = (tile / tp.nt[2]) % tp.nt[1], tx = tile / (tp.nt[2] * tp.nt[1]);
    const int o[3] = {tx * tp.T[0] - tp.lo, ty * tp.T[1] - tp.lo, tz * tp.T[2] - tp.lo};
    const size_t seg0 = (size_t)tile * m.S * tp.TV;
    if (cell_start[seg0] == cell_start[seg0 + (size_t)m.S * tp.TV]) return;   // empty tile (uniform)

    {
        uint4* z4 = reinterpret_cast<uint4*>(sm);
        const int n4 = (m.S * E3 + 3) / 4;
        for (int k = threadIdx.x; k < n4; k += SPREAD_THREADS) z4[k] = make_uint4(0u, 0u, 0u, 0u);
        if (threadIdx.x < EX) goff_x[threadIdx.x] = wrap_idx(o[0] + threadIdx.x, m.N[0]);
        else if (threadIdx.x >= 32 && threadIdx.x < 32 + EY) goff_y[threadIdx.x - 32] = wrap_idx(o[1] + threadIdx.x - 32, m.N[1]);
    }
    __syncthreads();

    // Lanes start their stencil on different x-planes (rotation by lane & 3): particles that share a cell, and so
    // every address, then hit different shared-memory banks in the same instruction instead of serialising.
    constexpr bool ROT = (P == 2 || P == 4);
    const int rot = ROT ? (int)(threadIdx.x & (P - 1)) : 0;
    uint32_t n_tile = 0;  // particles this thread accumulated through shared memory
    for (int sp = 0; sp < m.S; ++sp) {
        const uint32_t p_lo = cell_start[seg0 + (size_t)sp * tp.TV], p_hi = cell_start[seg0 + (size_t)(sp + 1) * tp.TV];
        uint32_t* ssp = sm + sp * E3;
        for (uint32_t i = p_lo + threadIdx.x; i < p_hi; i += SPREAD_THREADS) {
            int cell, b[3], d[3];
            float t, w[3][P];
            bool inside = true;
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                index_1d<P>(x[3 * (size_t)i + a], m.inv_h[a], cell, b[a], t);
                weights_1d<P>(t, w[a]);
                int dd = b[a] - o[a];            // in [-N, N+4]: one conditional wrap each way (N >= 8 here)
                dd += dd < 0 ? m.N[a] : 0;
                dd -= dd >= m.N[a] ? m.N[a] : 0;
                d[a] = dd;                        // local node of the stencil's first node (a periodic image)
                inside = inside && (dd + P <= (a == 2 ? EZ : EX));
            }
            if (inside) {
                uint32_t* s = ssp + (d[0] * EY + d[1]) * EZ + d[2];
#pragma unroll
                for (int k = 0; k < P; ++k) {
                    const int jx = ROT ? ((k + rot) & (P - 1)) : k;
                    float wx = w[0][0];
#pragma unroll
                    for (int q = 1; q < P; ++q) wx = (jx == q) ? w[0][q] : wx;
                    uint32_t* plane = s + jx * (EY * EZ);
#pragma unroll
                    for (int jy = 0; jy < P; ++jy) {
                        const float wxy = wx * w[1][jy];
#pragma unroll
                        for (int jz = 0; jz < P; ++jz)   // round(w 2^23) without F2I: mantissa of (w + 1), w in [0, 1]
                            atomicAdd(plane + jy * EZ + jz, __float_as_uint(fmaf(wxy, w[2][jz], 1.0f)) - 0x3F800000u);
                    }
                }
                ++n_tile;
            } else {
                // drifted out of the tile's halo since the last re-sort: rare, goes straight to the global grid
                spread_global_one<P>(m, b, w, grid + (size_t)sp * m.M, 1.0f);
            }
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
            const int sp = r / (EX * EY), q = r - sp * (EX * EY);
            const int lx = q / EY, ly = q - lx * EY;
            float* grow = grid + (size_t)sp * m.M + ((size_t)goff_x[lx] * m.N[1] + goff_y[ly]) * m.N[2];
            const uint32_t* srow = sm + r * EZ;
#pragma unroll
            for (int it = 0; it < (EZ + 31) / 32; ++it) {
                const int lz = lane + 32 * it;
                const uint32_t u = lz < EZ ? srow[lz] : 0u;
                if (u) {
                    if (pass == 0) tile_sum += u;
                    int gz = o[2] + lz;            // in [-lo, N + E): one conditional wrap each way
                    gz += gz < 0 ? m.N[2] : 0;
                    gz -= gz >= m.N[2] ? m.N[2] : 0;
                    atomicAdd(grow + gz, (float)u * sc);
                }
            }
        }
        if (pass == 1) break;
        const unsigned long long total = block_sum_u64(tile_sum, red);
        const unsigned long long cnt = block_sum_u64((unsigned long long)n_tile, red);
        const unsigned long long expect = cnt << FIX_BITS, slack = 64ull * cnt + 64ull;
        const bool ok = total + slack >= expect && total <= expect + slack;
        if (ok) return;                               // uniform across the block
    }
    // a node wrapped past 2^32 (>= 512 particles' worth on one node): redo this tile with fp32 global atomics
    for (int sp = 0; sp < m.S; ++sp) {
        const uint32_t p_lo = cell_start[seg0 + (size_t)sp * tp.TV], p_hi = cell_start[seg0 + (size_t)(sp + 1) * tp.TV];
        for (uint32_t i = p_lo + threadIdx.x; i < p_hi; i += SPREAD_THREADS) {
            int cell, b[3];
            float t, w[3][P];
            bool inside = true;
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                index_1d<P>(x[3 * (size_t)i + a], m.inv_h[a], cell, b[a], t);
                weights_1d<P>(t, w[a]);
                inside = inside && (wrap_idx(b[a] - o[a], m.N[a]) + P <= (a == 2 ? EZ : EX));
            }
            if (inside) spread_global_one<P>(m, b, w, grid + (size_t)sp * m.M, 1.0f);
        }
    }
}

// dispatch over (P, TZ): EZ = TZ + halo
template <int P, int TZ, typename F>
bool tile_case(int p, int tz, F&& f)
{
    if (p == P && tz == TZ) {
        f(spread_tile_kernel<P, TZ + ((P >= 3) ? 3 : 1)>);
        return true;
    }
    return false;
}
template <typename F>
bool tile_dispatch(int p, int tz, F&& f)
{
    return tile_case<1, 8>(p, tz, f) || tile_case<1, 16>(p, tz, f) || tile_case<1, 32>(p, tz, f) || tile_case<1, 64>(p, tz, f) ||
           tile_case<2, 8>(p, tz, f) || tile_case<2, 16>(p, tz, f) || tile_case<2, 32>(p, tz, f) || tile_case<2, 64>(p, tz, f) ||
           tile_case<3, 8>(p, tz, f) || tile_case<3, 16>(p, tz, f) || tile_case<3, 32>(p, tz, f) || tile_case<3, 64>(p, tz, f) ||
           tile_case<4, 8>(p, tz, f) || tile_case<4, 16>(p, tz, f) || tile_case<4, 32>(p, tz, f) || tile_case<4, 64>(p, tz, f);
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
    if (!c->tile.enabled) return TILD_OK;
    const size_t bytes = c->tile.smem_bytes;
    cudaError_t e = cudaSuccess;
    const bool found = tile_dispatch(c->mesh.P, c->tile.T[2], [&](auto kernel) {
        e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    });
    if (!found) return tild_fail(c, TILD_EINVAL, "no spread tile kernel for P=%d TZ=%d", c->mesh.P, c->tile.T[2]);
    if (e != cudaSuccess) return tild_fail(c, TILD_ECUDA, "cudaFuncSetAttribute(spread_tile_kernel, %zu B): %s", bytes, cudaGetErrorString(e));
    return TILD_OK;
}

// x must be sorted by (tile, species, cell) with cell_start = the counting-sort offsets of that key.
int launch_spread_tiled(tild_ctx* c, const uint32_t* cell_start, const float* x, float* grid)
{
    TILD_CUDA(c, cudaMemsetAsync(grid, 0, sizeof(float) * c->M * c->mesh.S, c->stream));
    if (c->mesh.n == 0) return TILD_OK;
    const TileParams& tp = c->tile;
    tile_dispatch(c->mesh.P, tp.T[2], [&](auto kernel) {
        kernel<<<tp.ntiles, SPREAD_THREADS, tp.smem_bytes, c->stream>>>(c->mesh, tp, cell_start, x, grid);
    });
    TILD_LAUNCH_CHECK(c, "spread_tile_kernel");
    return TILD_OK;
}
