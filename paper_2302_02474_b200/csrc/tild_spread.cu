// a2: particle -> mesh spread.  PAPER.md L223: "at each time-step, every particle assigns
// its density contribution to nearby grid points, using a spline interpolation scheme"; Eq. 1 L110.
// grid[J][g] = sum_{i in J} W_x W_y W_z  (raw weights), g = (ix*Ny + iy)*Nz + iz.
//
// Hot kernel: one CTA per tile of TX x TY x TZ cells (x a group of species).  The particles of the tile are one
// contiguous range of the segment-sorted arrays (tild_sort.cu).  The P^3 stencil of every particle is accumulated
// into a shared-memory image of the tile and the image is flushed to the global grid once, so global-atomic traffic
// is per tile node instead of per particle.
//
// Bank conflicts: 32 particles of a warp in cell order hit the 32 banks at random (measured 3.5 wavefronts per
// ATOMS, profiles/r1_before.md).  All P^3 stencil offsets are the same for every particle, so the bank
// of each access is (bank of the first stencil node) + const.  Each step the CTA therefore first bins its particles
// by that bank ("class") into 32 shared-memory lists (phase A: one shared atomic per particle), then works in rounds
// of one particle per class (phase B): lane c takes the k-th particle of class c, and every ATOMS of the round hits
// 32 different banks.  Binning every step makes this independent of how far particles drifted since the last re-sort.
//
// sm_100a has no native fp32 shared-memory atomic add (atomicAdd(float*) on shared compiles to an
// LDS + FADD + ATOMS.CAST.SPIN loop) but does have a native 32-bit integer one (ATOMS.ADD).  The tile is
// therefore accumulated in unsigned 2^-23 fixed point: each contribution is rounded once to 2^-23 (read off the
// bit pattern of the denormal w 2^-126, so no F2I on the XU pipe), the integer sum is exact and order-independent, and it is
// converted to fp32 at the flush.  A tile node holds < 512; a wrap is detected exactly by the tile's mass balance
// (sum of the tile == particles * 2^23 up to rounding) and such a tile is redone with fp32 global atomics.
#include "tild_internal.cuh"

namespace {

constexpr int SPREAD_THREADS = 512;
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
        inside = inside && ((unsigned)d[a] + (unsigned)P <= (unsigned)E[a]);   // unsigned: a wild position (d < 0) is not inside
    }
    return inside;
}

// weights only (the stencil position is already known): same single-rounded fp32 offsets as index_1d
template <int P>
__device__ __forceinline__ void offset_weights(const MeshParams& m, const float4& p, float w[3][P])
{
    const float pos[3] = {p.x, p.y, p.z};
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        int cell, b;
        float t;
        index_1d<P>(pos[a], m.inv_h[a], cell, b, t);
        weights_1d<P>(t, w[a]);
    }
}

// EY, EZ are template parameters so that every shared-memory offset of the stencil is an immediate.
// One CTA = one tile x one group of up to tp.sp_group species (blockIdx.y).
// Dynamic shared memory: image u32[nsp][EX][EY][EZ] | idx u32[KCAP][32] | ovf u32[CHUNK]; a list entry is
// (image word offset of the first stencil node << 12) | index of the particle in the chunk.
template <int P, int EY, int EZ>
__global__ void __launch_bounds__(SPREAD_THREADS, 2) spread_tile_kernel(MeshParams m, TileParams tp,
                                                                     const uint32_t* __restrict__ seg_base,
                                                                     const float4* __restrict__ X4, float* __restrict__ grid)
{
    constexpr int CHUNK = TILD_SPREAD_CHUNK, KCAP = TILD_SPREAD_KCAP;
    extern __shared__ __align__(16) uint32_t sm[];
    __shared__ unsigned long long red[SPREAD_WARPS];
    __shared__ int goff_x[32], goff_y[32];          // wrapped global x / y node of each local x / y
    __shared__ uint32_t cnt[32], novf, ndrift;
    __shared__ uint32_t rowoff[21 * 21];            // mesh offset of image row (lx, ly), z excluded
    const int EX = tp.E[0];
    const int E3 = EX * EY * EZ;
    const int tile = blockIdx.x;
    const int sp0 = blockIdx.y * tp.sp_group;
    const int nsp = min(tp.sp_group, m.S - sp0);
    const int tz = tile % tp.nt[2], ty = (tile / tp.nt[2]) % tp.nt[1], tx = tile / (tp.nt[2] * tp.nt[1]);
    const int o[3] = {tx * tp.T[0] - tp.lo, ty * tp.T[1] - tp.lo, tz * tp.T[2] - tp.lo - tp.sh};
    const int E[3] = {EX, tp.E[1], EZ};
    const size_t seg0 = (size_t)tile * m.S + sp0;
    const uint32_t p_lo = seg_base[seg0], p_hi = seg_base[seg0 + nsp];
    if (p_lo == p_hi) return;                        // empty tile (uniform)
    uint32_t* idx = sm + (size_t)tp.sp_group * E3;
    uint32_t* ovf = idx + KCAP * 32;

    {
        uint4* z4 = reinterpret_cast<uint4*>(sm);
        const int n4 = nsp * E3 / 4;                 // EZ % 4 == 0
        for (int k = threadIdx.x; k < n4; k += SPREAD_THREADS) z4[k] = make_uint4(0u, 0u, 0u, 0u);
        if (threadIdx.x < EX) goff_x[threadIdx.x] = wrap_idx(o[0] + threadIdx.x, m.N[0]);
        else if (threadIdx.x >= 32 && threadIdx.x < 32 + EY) goff_y[threadIdx.x - 32] = wrap_idx(o[1] + threadIdx.x - 32, m.N[1]);
        if (threadIdx.x < EX * EY) {                 // EX * EY <= 441 <= SPREAD_THREADS
            const int lx = threadIdx.x / EY, ly = threadIdx.x - lx * EY;
            rowoff[threadIdx.x] = (uint32_t)((wrap_idx(o[0] + lx, m.N[0]) * m.N[1] + wrap_idx(o[1] + ly, m.N[1])) * m.N[2]);
        }
    }
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    uint32_t n_tile = 0;  // particles this thread accumulated through shared memory

    for (uint32_t c0 = p_lo; c0 < p_hi; c0 += CHUNK) {
        const int nchunk = (int)min((uint32_t)CHUNK, p_hi - c0);
        // rounds reserved per class: a little above the mean; what does not fit is worked off in dense rounds of
        // mixed classes (a few bank conflicts) instead of rounds with idle lanes
        const uint32_t kcap = min((uint32_t)KCAP, (uint32_t)(nchunk + 31) / 32u + (uint32_t)(nchunk >> 9) + 1u);
        __syncthreads();                             // image zeroed / previous chunk's rounds done
        if (threadIdx.x < 32) cnt[threadIdx.x] = 0u;
        if (threadIdx.x == 32) novf = 0u;
        if (threadIdx.x == 33) ndrift = 0u;
        __syncthreads();
        // phase A: class of every particle = bank of its first stencil node in the image
        for (int i0 = threadIdx.x; i0 < nchunk; i0 += 4 * SPREAD_THREADS) {   // four loads in flight per thread
            float4 pj[4];
#pragma unroll
            for (int j = 0; j < 4; ++j)
                if (i0 + j * SPREAD_THREADS < nchunk) pj[j] = X4[c0 + i0 + j * SPREAD_THREADS];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
            const int i = i0 + j * SPREAD_THREADS;
            if (i >= nchunk) break;
            const float4 p = pj[j];
            const int spl = __float_as_int(p.w) - sp0;
            int b[3], d[3];
            float w[3][P];
            if (locate<P>(m, p, o, E, b, d, w)) {
                const uint32_t off = (uint32_t)(spl * E3 + (d[0] * EY + d[1]) * EZ + d[2]);
                const uint32_t cls = off & 31u, ent = (off << 12) | (uint32_t)i;
                const uint32_t k = atomicAdd(&cnt[cls], 1u);
                if (k < kcap) idx[k * 32 + cls] = ent;
                else ovf[atomicAdd(&novf, 1u)] = ent;
            } else {
                // drifted out of the tile's halo since the last re-sort: queued (from the top of ovf) and done
                // together after the rounds, so that one such particle does not stall the 31 other lanes here
                ovf[CHUNK - 1 - atomicAdd(&ndrift, 1u)] = (uint32_t)i;
            }
            }
        }
        __syncthreads();
        // phase B: rounds of one particle per class, then the overflow (any class)
        const uint32_t mine = cnt[lane];
        uint32_t rounds = mine;
#pragma unroll
        for (int dlt = 16; dlt > 0; dlt >>= 1) rounds = max(rounds, __shfl_xor_sync(0xffffffffu, rounds, dlt));
        rounds = min(rounds, kcap);
        const uint32_t extra = (novf + 31u) >> 5;
        for (uint32_t k = wid; k < rounds + extra; k += SPREAD_WARPS) {
            uint32_t ent = 0xFFFFFFFFu;
            if (k < rounds) {
                if (k < mine) ent = idx[k * 32 + lane];
            } else {
                const uint32_t j = (k - rounds) * 32u + lane;
                if (j < novf) ent = ovf[j];
            }
            if (ent == 0xFFFFFFFFu) continue;
            const float4 p = X4[c0 + (ent & 4095u)];
            float w[3][P];
            offset_weights<P>(m, p, w);
            uint32_t* s = sm + (ent >> 12);
            // round(w 2^23) with one FMUL and no F2I: w 2^-126 is a denormal (or the smallest normal for w = 1) whose
            // bit pattern IS the integer round(w 2^23); the two 2^-63 factors keep both operands normal, so the
            // product is rounded once, to nearest.  (Denormals are on: the library is built without -ftz.)
#pragma unroll
            for (int j = 0; j < P; ++j) {
                w[0][j] *= 0x1p-63f;
                w[2][j] *= 0x1p-63f;
            }
#pragma unroll
            for (int jx = 0; jx < P; ++jx) {
#pragma unroll
                for (int jy = 0; jy < P; ++jy) {
                    const float wxy = w[0][jx] * w[1][jy];
#pragma unroll
                    for (int jz = 0; jz < P; ++jz)
                        atomicAdd(s + (jx * EY + jy) * EZ + jz, __float_as_uint(__fmul_rn(wxy, w[2][jz])));
                }
            }
            ++n_tile;
        }
        // drifted particles of this chunk: straight to the global grid (fp32 reductions resolve in L2).  Kept in
        // this CTA: a separate kernel for them measured slower (its reductions no longer overlap other tiles' work)
        for (uint32_t j = threadIdx.x; j < ndrift; j += SPREAD_THREADS) {
            const float4 p = X4[c0 + ovf[CHUNK - 1 - j]];
            int b[3], d[3];
            float w[3][P];
            locate<P>(m, p, o, E, b, d, w);
            spread_global_one<P>(m, b, w, grid + (size_t)__float_as_int(p.w) * m.M);
        }
    }
    __syncthreads();

    // flush: consecutive threads take consecutive z of a row so that the global reductions are coalesced along z
    unsigned long long tile_sum = 0;
    constexpr int RPP = SPREAD_THREADS / EZ;               // rows per pass
    const int lz = threadIdx.x % EZ, r0 = threadIdx.x / EZ;
    const int gz = wrap_idx(o[2] + lz, m.N[2]);
    // 16-byte rows (Nz % 4 == 0: the image starts on a 16-byte boundary of the mesh rows, TileParams::sh, and every aligned
    // float4 of a row wraps as a whole): one vector reduction (red.global.add.v4.f32, REDG.E.ADD.F32x4) per four nodes
    static_assert(EZ % 4 == 0, "image rows are whole float4s");
    const bool vec4 = m.N[2] % 4 == 0 && (reinterpret_cast<uintptr_t>(grid) & 15) == 0 && (m.M % 4) == 0;
    for (int pass = 0; pass < 2; ++pass) {          // pass 1 only runs to undo a wrapped tile
        const float sc = pass == 0 ? FIX_INV : -FIX_INV;
        if (vec4) {
            constexpr int CPR = EZ / 4, RPP4 = SPREAD_THREADS / CPR;
            const int c4 = threadIdx.x % CPR, rr = threadIdx.x / CPR;
            const int gz4 = wrap_idx(o[2] + 4 * c4, m.N[2]);
            if (rr < RPP4) {
                for (int spl = 0; spl < nsp; ++spl) {
                    float* gsp = grid + (size_t)(sp0 + spl) * m.M + gz4;
                    const uint4* simg = reinterpret_cast<const uint4*>(sm + spl * E3) + c4;
                    for (int q = rr; q < EX * EY; q += RPP4) {
                        const uint4 u = simg[q * CPR];
                        if (u.x | u.y | u.z | u.w) {
                            if (pass == 0) tile_sum += (unsigned long long)u.x + u.y + u.z + u.w;
                            asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(gsp + rowoff[q]), "f"((float)u.x * sc),
                                         "f"((float)u.y * sc), "f"((float)u.z * sc), "f"((float)u.w * sc)
                                         : "memory");
                        }
                    }
                }
            }
        } else if (r0 < RPP) {
            for (int spl = 0; spl < nsp; ++spl) {
                float* gsp = grid + (size_t)(sp0 + spl) * m.M + gz;
                const uint32_t* simg = sm + spl * E3 + lz;
                for (int q = r0; q < EX * EY; q += RPP) {
                    const uint32_t u = simg[q * EZ];
                    if (u) {
                        if (pass == 0) tile_sum += u;
                        atomicAdd(gsp + rowoff[q], (float)u * sc);
                    }
                }
            }
        }
        if (pass == 1) break;
        // A node can only wrap past 2^32 if >= 2^9 / (largest single-node weight) particles sit on it: the largest
        // weight is 1 (P <= 2), (3/4)^3 (P = 3), (23/48)^3 (P = 4).  Tiles with fewer particles skip the check.
        constexpr uint32_t SAFE = P <= 2 ? 511u : (P == 3 ? 1213u : (P == 4 ? 4653u : 2381u));   // P = 5: (115/192)^3
        if (p_hi - p_lo <= SAFE) return;              // uniform across the block
        const unsigned long long total = block_sum_u64(tile_sum, red);
        const unsigned long long cntp = block_sum_u64((unsigned long long)n_tile, red);
        const unsigned long long expect = cntp << FIX_BITS, slack = 64ull * cntp + 64ull;
        const bool ok = total + slack >= expect && total <= expect + slack;
        if (ok) return;                               // uniform across the block
    }
    // a node wrapped past 2^32 (>= 512 particles' worth on one node): redo this tile with fp32 global atomics
    for (uint32_t i = p_lo + threadIdx.x; i < p_hi; i += SPREAD_THREADS) {
        const float4 p = X4[i];
        int b[3], d[3];
        float w[3][P];
        if (locate<P>(m, p, o, E, b, d, w)) spread_global_one<P>(m, b, w, grid + (size_t)__float_as_int(p.w) * m.M);
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
    constexpr int H = Halo<P>::H, EZA = Halo<P>::EZA, EZB = Halo<P>::EZB;
    return tile_case<P, 8 + H, EZA>(p, ey, ez, f) || tile_case<P, 8 + H, EZB>(p, ey, ez, f) ||
           tile_case<P, 16 + H, EZA>(p, ey, ez, f) || tile_case<P, 16 + H, EZB>(p, ey, ez, f);
}
template <typename F>
bool tile_dispatch(int p, int ey, int ez, F&& f)
{
    return tile_dispatch_p<1>(p, ey, ez, f) || tile_dispatch_p<2>(p, ey, ez, f) || tile_dispatch_p<3>(p, ey, ez, f) ||
           tile_dispatch_p<4>(p, ey, ez, f) || tile_dispatch_p<5>(p, ey, ez, f);
}

int spread_slots(tild_ctx* c, size_t s0, size_t s1, const float4* X4, float* grid)
{
    if (s1 <= s0) return TILD_OK;
    const unsigned nb = (unsigned)((s1 - s0 + 255) / 256);
    switch (c->mesh.P) {
    case 1: spread_slots_kernel<1><<<nb, 256, 0, c->stream>>>(c->mesh, s0, s1, X4, grid); break;
    case 2: spread_slots_kernel<2><<<nb, 256, 0, c->stream>>>(c->mesh, s0, s1, X4, grid); break;
    case 3: spread_slots_kernel<3><<<nb, 256, 0, c->stream>>>(c->mesh, s0, s1, X4, grid); break;
    case 4: spread_slots_kernel<4><<<nb, 256, 0, c->stream>>>(c->mesh, s0, s1, X4, grid); break;
    default: spread_slots_kernel<5><<<nb, 256, 0, c->stream>>>(c->mesh, s0, s1, X4, grid); break;
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
        e = tild_raise_smem_limit(reinterpret_cast<const void*>(kernel), bytes);
    });
    if (found && e == cudaSuccess && spread_rot_applies(c)) e = spread_rot_run(c, nullptr, nullptr, nullptr, true);
    if (!found) return tild_fail(c, TILD_EINVAL, "no spread tile kernel for P=%d EY=%d EZ=%d", c->mesh.P, c->tile.EY, c->tile.EZ);
    if (e != cudaSuccess) return tild_fail(c, TILD_ECUDA, "cudaFuncSetAttribute(spread_tile_kernel, %zu B): %s", bytes, cudaGetErrorString(e));
    return TILD_OK;
}

// X4 must be segment-sorted with the offsets lay.seg_base.
int launch_spread(tild_ctx* c, const SegLayout& lay, const float4* X4, float* grid)
{
    // the library's own grid comes back cleared from the fused step (interp_drift_kernel); anything else is cleared here
    if (!(grid == c->grid && c->grid_clean)) TILD_CUDA(c, cudaMemsetAsync(grid, 0, sizeof(float) * c->M * c->mesh.S, c->stream));
    if (grid == c->grid) c->grid_clean = false;
    if (c->mesh.n == 0) {
        if (grid == c->grid) c->grid_clean = true;
        return TILD_OK;
    }
    const TileParams& tp = c->tile;
    // P = 1 touches one node per particle: the per-particle kernel is faster than any tiling (profiles/r1_c5_sweep.md)
    if (!tp.enabled || c->mesh.P == 1 || (c->prm.flags & TILD_FLAG_NAIVE_SPREAD)) return spread_slots(c, 0, (size_t)c->mesh.n, X4, grid);
    if (spread_rot_applies(c) && !(c->prm.flags & TILD_FLAG_GEN1_TILES)) {
        spread_rot_run(c, lay.seg_base, X4, grid, false);
        TILD_LAUNCH_CHECK(c, "spread_rot_kernel");
        return TILD_OK;
    }
    const dim3 g((unsigned)tp.ntiles, (unsigned)((c->mesh.S + tp.sp_group - 1) / tp.sp_group));
    tile_dispatch(c->mesh.P, tp.EY, tp.EZ, [&](auto kernel) {
        kernel<<<g, SPREAD_THREADS, tp.smem_spread, c->stream>>>(c->mesh, tp, lay.seg_base, X4, grid);
    });
    TILD_LAUNCH_CHECK(c, "spread_tile_kernel");
    return TILD_OK;
}
