// a2: particle -> mesh spread.  PAPER.md L223: "at each time-step, every particle assigns
// its density contribution to nearby grid points, using a spline interpolation scheme"; Eq. 1 L110.
// grid[J][g] = sum_{i in J} W_x W_y W_z  (raw weights), g = (ix*Ny + iy)*Nz + iz.
//
// Hot kernel: one CTA per tile of TX x TY x TZ cells.  The particles of the tile sit in the slab-transposed
// layout of tild_sort.cu: a warp reads one round (32 consecutive slots, one coalesced 512-byte load) in which lane r
// holds a particle whose z cell is r mod 32.  The P^3 stencil of every particle is accumulated into a shared-memory
// image of the tile whose z extent EZ is a multiple of 32, so the bank of a stencil node is (r + const) mod 32:
// every shared-memory atomic of a warp instruction hits 32 different banks.  (With particles in plain cell order
// the same kernel measured 3.5 wavefronts per ATOMS; profiles/r1_before_slab_layout.md.)  The tile is flushed to the
// global grid once, so global-atomic traffic is per tile node instead of per particle.
//
// sm_100a has no native fp32 shared-memory atomic add (atomicAdd(float*) on shared compiles to an
// LDS + FADD + ATOMS.CAST.SPIN loop) but does have a native 32-bit integer one (ATOMS.ADD).  The tile is
// therefore accumulated in unsigned 2^-23 fixed point: each contribution is rounded once to 2^-23 (read off the
// mantissa of 1 + w, so no F2I on the XU pipe), the integer sum is exact and order-independent, and it is
// converted to fp32 at the flush.  A tile node holds < 512; a wrap is detected exactly by the tile's mass balance
// (sum of the tile == particles * 2^23 up to rounding) and such a tile is redone with fp32 global atomics.
#include "tild_internal.cuh"

namespace {

constexpr int SPREAD_THREADS = 256;
constexpr int SPREAD_WARPS = SPREAD_THREADS / 32;
constexpr int FIX_BITS = 23;                    // tile fixed point: units of 2^-23
constexpr float FIX_INV = 1.0f / 8388608.0f;

// Baseline / fallback: one thread per particle, P^3 global reductions (REDG.E.ADD.F32 resolves in L2).
template <int P>
__device__ __forceinline__ void spread_global_one(const MeshParams& m, const int b[3], const float w[3][P], float* __restrict__ g)
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
            const float wxy = w[0][jx] * w[1][jy];
#pragma unroll
            for (int jz = 0; jz < P; ++jz) atomicAdd(g + row + iz[jz], wxy * w[2][jz]);
        }
    }
}

// per-particle kernel over the slots [s0, s1): the overflow tail, or everything when the tile kernel is disabled
template <int P>
__global__ void __launch_bounds__(256) spread_slots_kernel(MeshParams m, size_t s0, size_t s1, const float4* __restrict__ X4,
                                                           float* __restrict__ grid)
{
    const size_t s = s0 + (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= s1) return;
    const float4 p = X4[s];
    const int type = __float_as_int(p.w);
    if (type < 0) return;
    const float pos[3] = {p.x, p.y, p.z};
    int cell, b[3];
    float t, w[3][P];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        index_1d<P>(pos[a], m.inv_h[a], cell, b[a], t);
        weights_1d<P>(t, w[a]);
    }
    spread_global_one<P>(m, b, w, grid + (size_t)type * m.M);
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
    for (int k = 0; k < SPREAD_WARPS; ++k) s += scratch[k];
    return s;
}

// index map + weights of one particle and the local (shared-memory) coordinates of its first stencil node
template <int P>
__device__ __forceinline__ bool locate(const MeshParams& m, const float4& p, const int o[3], const int E[3], int b[3], int d[3],
                                       float w[3][P])
{
    const float pos[3] = {p.x, p.y, p.z};
    bool inside = true;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        int cell;
        float t;
        index_1d<P>(pos[a], m.inv_h[a], cell, b[a], t);
        weights_1d<P>(t, w[a]);
        d[a] = wrap_near(b[a] - o[a], m.N[a]);  // a periodic image of the stencil's first node, relative to the tile (N >= 8)
        inside = inside && (d[a] + P <= E[a]);
    }
    return inside;
}

// EY, EZ are template parameters so that every shared-memory offset of the stencil is an immediate.
// One CTA = one tile x one group of up to tp.sp_group species (blockIdx.y).
template <int P, int EY, int EZ>
__global__ void __launch_bounds__(SPREAD_THREADS) spread_tile_kernel(MeshParams m, TileParams tp,
                                                                     const uint32_t* __restrict__ seg_base,
                                                                     const float4* __restrict__ X4, float* __restrict__ grid)
{
    extern __shared__ __align__(16) uint32_t sm[];
    __shared__ unsigned long long red[SPREAD_WARPS];
    __shared__ int goff_x[32], goff_y[32];          // wrapped global x / y node of each local x / y
    __shared__ uint32_t sbase[TILD_MAX_SPECIES + 1], srounds[TILD_MAX_SPECIES + 1];
    const int EX = tp.E[0];
    const int E3 = EX * EY * EZ;
    const int tile = blockIdx.x;
    const int sp0 = blockIdx.y * tp.sp_group;
    const int nsp = min(tp.sp_group, m.S - sp0);
    const int tz = tile % tp.nt[2], ty = (tile / tp.nt[2]) % tp.nt[1], tx = tile / (tp.nt[2] * tp.nt[1]);
    const int o[3] = {tx * tp.T[0] - tp.lo, ty * tp.T[1] - tp.lo, tz * tp.T[2] - tp.lo - tp.sh};
    const int E[3] = {EX, tp.E[1], EZ};
    const size_t seg0 = (size_t)tile * m.S + sp0;
    if (seg_base[seg0] == seg_base[seg0 + nsp]) return;   // empty tile (uniform)

    {
        uint4* z4 = reinterpret_cast<uint4*>(sm);
        const int n4 = nsp * E3 / 4;                 // EZ % 32 == 0
        for (int k = threadIdx.x; k < n4; k += SPREAD_THREADS) z4[k] = make_uint4(0u, 0u, 0u, 0u);
        if (threadIdx.x < EX) goff_x[threadIdx.x] = wrap_idx(o[0] + threadIdx.x, m.N[0]);
        else if (threadIdx.x >= 32 && threadIdx.x < 32 + EY) goff_y[threadIdx.x - 32] = wrap_idx(o[1] + threadIdx.x - 32, m.N[1]);
        if (threadIdx.x == 64) {                     // prefix of the rounds of this CTA's segments
            uint32_t acc = 0;
            for (int sp = 0; sp < nsp; ++sp) {
                srounds[sp] = acc;
                sbase[sp] = seg_base[seg0 + sp];
                acc += (seg_base[seg0 + sp + 1] - sbase[sp]) >> 5;
            }
            srounds[nsp] = acc;
        }
    }
    __syncthreads();

    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    uint32_t n_tile = 0;  // particles this thread accumulated through shared memory
    const uint32_t rounds_total = srounds[nsp];
    int sp = 0;
    for (uint32_t j = wid; j < rounds_total; j += SPREAD_WARPS) {
        while (j >= srounds[sp + 1]) ++sp;           // warp-uniform
        const float4 p = X4[(size_t)sbase[sp] + (size_t)(j - srounds[sp]) * 32u + lane];
        if (__float_as_int(p.w) < 0) continue;       // hole
        int b[3], d[3];
        float w[3][P];
        if (locate<P>(m, p, o, E, b, d, w)) {
            uint32_t* s = sm + sp * E3 + (d[0] * EY + d[1]) * EZ + d[2];
#pragma unroll
            for (int jx = 0; jx < P; ++jx) {
#pragma unroll
                for (int jy = 0; jy < P; ++jy) {
                    const float wxy = w[0][jx] * w[1][jy];
#pragma unroll
                    for (int jz = 0; jz < P; ++jz)       // round(w 2^23) without F2I: mantissa of (w + 1), w in [0, 1]
                        atomicAdd(s + (jx * EY + jy) * EZ + jz, __float_as_uint(fmaf(wxy, w[2][jz], 1.0f)) - 0x3F800000u);
                }
            }
            ++n_tile;
        } else {
            // drifted out of the tile's halo since the last re-sort: rare, goes straight to the global grid
            spread_global_one<P>(m, b, w, grid + (size_t)(sp0 + sp) * m.M);
        }
    }
    __syncthreads();

    // flush: one warp per z-row of the tile so that the global reductions are coalesced along z
    unsigned long long tile_sum = 0;
    int gz[EZ / 32];
#pragma unroll
    for (int it = 0; it < EZ / 32; ++it) gz[it] = wrap_idx(o[2] + lane + 32 * it, m.N[2]);
    for (int pass = 0; pass < 2; ++pass) {          // pass 1 only runs to undo a wrapped tile
        const float sc = pass == 0 ? FIX_INV : -FIX_INV;
        for (int spl = 0; spl < nsp; ++spl) {
            float* gsp = grid + (size_t)(sp0 + spl) * m.M;
            for (int q = wid; q < EX * EY; q += SPREAD_WARPS) {
                const int lx = q / EY, ly = q - lx * EY;
                if (ly >= E[1]) continue;
                float* grow = gsp + ((size_t)goff_x[lx] * m.N[1] + goff_y[ly]) * m.N[2];
                const uint32_t* srow = sm + (spl * EX * EY + q) * EZ + lane;
#pragma unroll
                for (int it = 0; it < EZ / 32; ++it) {
                    const uint32_t u = srow[32 * it];
                    if (u) {
                        if (pass == 0) tile_sum += u;
                        atomicAdd(grow + gz[it], (float)u * sc);
                    }
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
    sp = 0;
    for (uint32_t j = wid; j < rounds_total; j += SPREAD_WARPS) {
        while (j >= srounds[sp + 1]) ++sp;
        const float4 p = X4[(size_t)sbase[sp] + (size_t)(j - srounds[sp]) * 32u + lane];
        if (__float_as_int(p.w) < 0) continue;
        int b[3], d[3];
        float w[3][P];
        if (locate<P>(m, p, o, E, b, d, w)) spread_global_one<P>(m, b, w, grid + (size_t)(sp0 + sp) * m.M);
    }
}

// dispatch over (P, EY, EZ); EY in {9, 17} for P <= 2 and {11, 19} for P >= 3 (tile edge 8 or 16 + halo)
template <int P, int EY, int EZ, typename F>
bool tile_case(int p, int ey, int ez, F&& f)
{
    if (p == P && ey == EY && ez == EZ) {
        f(spread_tile_kernel<P, EY, EZ>);
        return true;
    }
    return false;
}
template <int P, typename F>
bool tile_dispatch_p(int p, int ey, int ez, F&& f)
{
    constexpr int H = (P >= 3) ? 3 : 1;
    return tile_case<P, 8 + H, 32>(p, ey, ez, f) || tile_case<P, 8 + H, 64>(p, ey, ez, f) ||
           tile_case<P, 16 + H, 32>(p, ey, ez, f) || tile_case<P, 16 + H, 64>(p, ey, ez, f);
}
template <typename F>
bool tile_dispatch(int p, int ey, int ez, F&& f)
{
    return tile_dispatch_p<1>(p, ey, ez, f) || tile_dispatch_p<2>(p, ey, ez, f) || tile_dispatch_p<3>(p, ey, ez, f) ||
           tile_dispatch_p<4>(p, ey, ez, f);
}

int spread_slots(tild_ctx* c, size_t s0, size_t s1, const float4* X4, float* grid)
{
    if (s1 <= s0) return TILD_OK;
    const unsigned nb = (unsigned)((s1 - s0 + 255) / 256);
    switch (c->mesh.P) {
    case 1: spread_slots_kernel<1><<<nb, 256, 0, c->stream>>>(c->mesh, s0, s1, X4, grid); break;
    case 2: spread_slots_kernel<2><<<nb, 256, 0, c->stream>>>(c->mesh, s0, s1, X4, grid); break;
    case 3: spread_slots_kernel<3><<<nb, 256, 0, c->stream>>>(c->mesh, s0, s1, X4, grid); break;
    default: spread_slots_kernel<4><<<nb, 256, 0, c->stream>>>(c->mesh, s0, s1, X4, grid); break;
    }
    TILD_LAUNCH_CHECK(c, "spread_slots_kernel");
    return TILD_OK;
}

}  // namespace

int tild_spread_configure(tild_ctx* c)
{
    if (!c->tile.enabled) return TILD_OK;
    const size_t bytes = c->tile.smem_spread;
    cudaError_t e = cudaSuccess;
    const bool found = tile_dispatch(c->mesh.P, c->tile.EY, c->tile.EZ, [&](auto kernel) {
        e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    });
    if (!found) return tild_fail(c, TILD_EINVAL, "no spread tile kernel for P=%d EY=%d EZ=%d", c->mesh.P, c->tile.EY, c->tile.EZ);
    if (e != cudaSuccess) return tild_fail(c, TILD_ECUDA, "cudaFuncSetAttribute(spread_tile_kernel, %zu B): %s", bytes, cudaGetErrorString(e));
    return TILD_OK;
}

// X4 must be in the slab-transposed layout described by lay.
int launch_spread(tild_ctx* c, const EllLayout& lay, const float4* X4, float* grid)
{
    TILD_CUDA(c, cudaMemsetAsync(grid, 0, sizeof(float) * c->M * c->mesh.S, c->stream));
    if (c->mesh.n == 0) return TILD_OK;
    const TileParams& tp = c->tile;
    if (tp.enabled && lay.total_ell > 0) {
        const dim3 g((unsigned)tp.ntiles, (unsigned)((c->mesh.S + tp.sp_group - 1) / tp.sp_group));
        tile_dispatch(c->mesh.P, tp.EY, tp.EZ, [&](auto kernel) {
            kernel<<<g, SPREAD_THREADS, tp.smem_spread, c->stream>>>(c->mesh, tp, lay.seg_base, X4, grid);
        });
        TILD_LAUNCH_CHECK(c, "spread_tile_kernel");
    }
    return spread_slots(c, lay.total_ell, lay.used(), X4, grid);
}
