// a2, cubic assignment (P = 4): particle -> mesh spread (Eq. 1, Fig. 1),
// second-generation tile kernel.  Same shared-memory fixed-point tile image and mass-balance wrap check as
// tild_spread.cu; what changes is how the particles reach the image:
//
//  * Rotation groups (see tild_interp_rot.cu): with EZ = 8 or 24 mod 32 the four y rows of a stencil start 0, 8, 16, 24
//    banks apart, so traversing them in the order (jy + r) mod 4 moves a particle from bank class c to c + 8r.  A
//    particle fits any of the four lanes g, g+8, g+16, g+24 (g = c mod 8): 8 groups filled round-robin instead of 32
//    classes with overflow rounds, and every ATOMS of a round hits 32 different banks.
//  * The list entry carries the three stencil offsets (25-bit fixed point), the image offset and the rotation in 12 bytes
//    of shared memory.  The rounds read nothing from global memory: with the whole L1 carved out as shared memory the
//    first-generation kernel's re-load of every position in class order was an L2 round trip per particle.
#include "tild_internal.cuh"

#include <type_traits>

namespace {

#ifndef TILD_SROT_SCALAR_FLUSH
#define TILD_SROT_SCALAR_FLUSH 0   // 1: one scalar RED per node also where the vector reduction applies (A/B)
#endif
#ifndef TILD_SROT_FMUL2
#define TILD_SROT_FMUL2 1   // packed FMUL2 for the 64 weight products of a particle (0.2291 -> 0.2277 ms on C4)
#endif
#ifndef TILD_SROT_THREADS
// chunk of 3072 > the ~2048 particles of a C4 tile: a tile just above a chunk of 2048 was split into two chunks of ~1030,
// whose 33-36 rounds fill the 16 warps' third turn only to a fifth (spread 0.2277 -> 0.2135 ms)
#define TILD_SROT_THREADS 512
#define TILD_SROT_CHUNK 3072
#define TILD_SROT_KCAP 110
#endif
constexpr int ST = TILD_SROT_THREADS;   // threads per CTA
constexpr int SW = ST / 32;
constexpr int SCHUNK = TILD_SROT_CHUNK; // particles binned at a time (all species of the CTA's group)
constexpr int SPT = SCHUNK / ST;        // particles per thread and chunk
constexpr int SKCAP = TILD_SROT_KCAP;   // rounds of list space (mean SCHUNK / 32 for a full chunk)
constexpr int SSLOTS = SKCAP * 32;
constexpr int SEX = 11;                 // image edge in x: 8 cells + halo 3
constexpr int SDCAP = 256;              // drifted particles per chunk queued for dense processing
constexpr int FIX_BITS = 23;            // tile fixed point: units of 2^-23
constexpr float FIX_INV = 1.0f / 8388608.0f;

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

// one particle straight to the global grid (fp32 reductions resolve in L2): drifted particles, wrapped tiles
__device__ __forceinline__ void spread_particle_global(const MeshParams& m, const float4& p, float* __restrict__ grid)
{
    const float pos[3] = {p.x, p.y, p.z};
    int b[3];
    float w[3][4];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        int cell;
        float t;
        index_1d<4>(pos[a], m.inv_h[a], cell, b[a], t);
        weights_1d<4>(t, w[a]);
    }
    spread_global_one<4>(m, b, w, grid + (size_t)__float_as_int(p.w) * m.M);
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
    for (int k = 0; k < SW; ++k) s += scratch[k];
    return s;
}

// One CTA = one tile x one group of up to sp_group species.  Grid (nt_z, nt_y, nt_x x groups): the tile coordinates are the
// block indices (no integer divisions in the prologue of 4096 x 16 warps), launch order = linear tile order.
// Dynamic shared memory: image u32[sp_group][SEX][EY][EZ] | ent u32[3][SSLOTS].
template <int EY, int EZ>
__global__ void __launch_bounds__(ST, 2) spread_rot_kernel(MeshParams m, TileParams tp, int sp_group, const uint32_t* __restrict__ seg_base,
                                                          const float4* __restrict__ X4, float* __restrict__ grid)
{
    constexpr int P = 4, E3 = SEX * EY * EZ;
    static_assert(EZ % 32 == 8 || EZ % 32 == 24, "row rotation needs the P rows of a stencil to tile the 32 banks");
    extern __shared__ __align__(16) uint32_t sm[];
    __shared__ unsigned long long red[SW];
    __shared__ uint32_t gcnt[2][8], nq[2];
    __shared__ uint16_t dq[SDCAP];                  // drifted particles of the chunk, done densely after the rounds
    __shared__ uint32_t rowoff[SEX * EY];           // mesh offset of image row (lx, ly), z excluded
    const int tz = blockIdx.x, ty = blockIdx.y;
    int tx = blockIdx.z, grp = 0;
    if (sp_group < m.S) {                            // more than one species group (uniform): blockIdx.z = group * nt_x + tx
        grp = tx / tp.nt[0];
        tx -= grp * tp.nt[0];
    }
    const int tile = (tx * tp.nt[1] + ty) * tp.nt[2] + tz;
    const int sp0 = grp * sp_group;
    const int nsp = min(sp_group, m.S - sp0);
    const int o[3] = {tx * tp.T[0] - tp.lo, ty * tp.T[1] - tp.lo, tz * tp.T[2] - tp.lo - tp.sh};
    const int E[3] = {SEX, tp.E[1], EZ};
    const size_t seg0 = (size_t)tile * m.S + sp0;
    const uint32_t p_lo = seg_base[seg0], p_hi = seg_base[seg0 + nsp];   // used after the first half of the zeroing: their
                                                                         // L2 / DRAM round trip runs under it
    uint32_t* ent = sm + (size_t)sp_group * E3;
    uint4* z4 = reinterpret_cast<uint4*>(sm);
    const int n4 = nsp * E3 / 4;                     // EZ % 4 == 0
    const int n4a = (n4 / 2 + ST - 1) / ST * ST;     // first half: whole passes of the CTA
    for (int k = threadIdx.x; k < min(n4a, n4); k += ST) z4[k] = make_uint4(0u, 0u, 0u, 0u);
    if (p_lo == p_hi) return;                        // empty tile (uniform)
    // the tile's positions on their way to L2 while the rest of the image is zeroed (8 particles per 128-byte line)
    for (uint32_t i = p_lo + 8u * threadIdx.x; i < p_hi; i += 8u * ST) asm volatile("prefetch.global.L2 [%0];" ::"l"(X4 + i));
    {
        for (int k = n4a + threadIdx.x; k < n4; k += ST) z4[k] = make_uint4(0u, 0u, 0u, 0u);
        if (threadIdx.x < SEX * EY) {
            const int lx = threadIdx.x / EY, ly = threadIdx.x - lx * EY;
            rowoff[threadIdx.x] = (uint32_t)((wrap_idx(o[0] + lx, m.N[0]) * m.N[1] + wrap_idx(o[1] + ly, m.N[1])) * m.N[2]);
        }
        if (threadIdx.x < 16) gcnt[threadIdx.x >> 3][threadIdx.x & 7] = 0u;
        if (threadIdx.x == 16) nq[0] = nq[1] = 0u;
    }
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    uint32_t n_tile = 0;                             // particles this thread accumulated through shared memory
    uint32_t per = (p_hi - p_lo + SCHUNK - 1) / SCHUNK;
    per = ((p_hi - p_lo + per - 1) / per + 31u) & ~31u;            // equal chunks, whole rounds
    __syncthreads();                                 // image zeroed, counters visible
    int par = 0;
    for (uint32_t c0 = p_lo; c0 < p_hi; c0 += per, par ^= 1) {
        const int nchunk = (int)min(per, p_hi - c0);
        if (threadIdx.x < 8) gcnt[par ^ 1][threadIdx.x] = 0u;     // the next chunk's counters (last read two barriers ago)
        if (threadIdx.x == 8) nq[par ^ 1] = 0u;
        // ---- phase A: bin by rotation group ------------------------------------------------------------------------
#ifdef TILD_SROT_BATCH
        float4 pa[SPT];
#pragma unroll
        for (int j = 0; j < SPT; ++j)
            if (threadIdx.x + j * ST < nchunk) pa[j] = X4[(size_t)c0 + threadIdx.x + j * ST];
#endif
#ifndef TILD_SROT_BATCH
        // one load ahead: the position of particle j + 1 is on its way while particle j is binned
        float4 pnext = make_float4(0.f, 0.f, 0.f, 0.f);
        if ((int)threadIdx.x < nchunk) pnext = X4[(size_t)c0 + threadIdx.x];
#endif
#pragma unroll
        for (int j = 0; j < SPT; ++j) {
            if (threadIdx.x + j * ST >= nchunk) break;       // later j are beyond the chunk too
#ifdef TILD_SROT_BATCH
            const float4 p = pa[j];
#else
            const float4 p = pnext;
            if (j + 1 < SPT && threadIdx.x + (j + 1) * ST < nchunk) pnext = X4[(size_t)c0 + threadIdx.x + (j + 1) * ST];
#endif
            const float pos[3] = {p.x, p.y, p.z};
            int d[3];
            float t[3];
            bool inside = true;
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                int cell, b;
                index_1d<P>(pos[a], m.inv_h[a], cell, b, t[a]);
                d[a] = wrap_near(b - o[a], m.N[a]);
                inside = inside && ((unsigned)d[a] + (unsigned)P <= (unsigned)E[a]);   // unsigned: a wild position (d < 0) is not inside
            }
            uint32_t k = SKCAP, pos4 = 0, off = 0;
            if (inside) {
                off = (uint32_t)((__float_as_int(p.w) - sp0) * E3 + (d[0] * EY + d[1]) * EZ + d[2]);
                pos4 = atomicAdd(&gcnt[par][off & 7u], 1u);
                k = pos4 >> 2;
            }
            if (k < SKCAP) {
                const uint32_t ln = (off & 7u) + 8u * (pos4 & 3u);    // lane that will take it
                const uint32_t r = ((EZ % 32 == 8 ? ln - off : off - ln) >> 3) & 3u;   // rows traversed as (jy + r) mod 4
                const uint32_t slot = k * 32u + ln;
                const int q0 = __float2int_rn(t[0] * 16777216.0f), q1 = __float2int_rn(t[1] * 16777216.0f),
                          q2 = __float2int_rn(t[2] * 16777216.0f);
                ent[slot] = ((uint32_t)q0 & 0x1FFFFFFu) | (off << 25);                       // off bits 0..6
                ent[SSLOTS + slot] = ((uint32_t)q1 & 0x1FFFFFFu) | ((off >> 7) << 25);        // off bits 7..13
                ent[2 * SSLOTS + slot] = ((uint32_t)q2 & 0x1FFFFFFu) | (((off >> 14) & 31u) << 25) | (r << 30);
            } else {
                // left the tile's image since the last re-sort (or no list space): straight to the global grid, queued so
                // that one such particle does not stall the 31 other lanes here
                const uint32_t dj = atomicAdd(&nq[par], 1u);
                if (dj < (uint32_t)SDCAP) dq[dj] = (uint16_t)(threadIdx.x + j * ST);
                else spread_particle_global(m, p, grid);
            }
        }
        __syncthreads();
        // ---- rounds: lane l takes the k-th quadruple of group l & 7 --------------------------------------------------
        const uint32_t mine = min(gcnt[par][lane & 7], (uint32_t)(4 * SKCAP));
        uint32_t rounds = mine;
#pragma unroll
        for (int dlt = 4; dlt > 0; dlt >>= 1) rounds = max(rounds, __shfl_xor_sync(0xffffffffu, rounds, dlt));
        rounds = (rounds + 3u) >> 2;
        for (uint32_t k = wid; k < rounds; k += SW) {
            if (4u * k + (uint32_t)(lane >> 3) >= mine) continue;
            const uint32_t slot = k * 32u + lane;
            const uint32_t e0 = ent[slot], e1 = ent[SSLOTS + slot], e2 = ent[2 * SSLOTS + slot];
            const float tx_ = (float)((int)(e0 << 7) >> 7) * (1.0f / 16777216.0f);
            const float ty_ = (float)((int)(e1 << 7) >> 7) * (1.0f / 16777216.0f);
            const float tz_ = (float)((int)(e2 << 7) >> 7) * (1.0f / 16777216.0f);
            const uint32_t off = (e0 >> 25) | ((e1 >> 25) << 7) | (((e2 >> 25) & 31u) << 14), r = e2 >> 30;
            float wx[P], wy[P], wz[P];
            weights_1d<P>(tx_, wx);
            weights_1d<P>(ty_, wy);
            weights_1d<P>(tz_, wz);
            // round(w 2^23) with one FMUL and no F2I: w 2^-126 is a denormal (or the smallest normal for w = 1) whose
            // bit pattern IS the integer round(w 2^23); the two 2^-63 factors keep both operands normal, so the
            // product is rounded once, to nearest.  (Denormals are on: the library is built without -ftz.)
#pragma unroll
            for (int j = 0; j < P; ++j) {
                wx[j] *= 0x1p-63f;
                wz[j] *= 0x1p-63f;
            }
            uint32_t* row[P];
            float wyr[P];
            {
                const bool r1 = r & 1u, r2 = r & 2u;
                const float b0 = r1 ? wy[1] : wy[0], b1 = r1 ? wy[2] : wy[1], b2 = r1 ? wy[3] : wy[2], b3 = r1 ? wy[0] : wy[3];
                wyr[0] = r2 ? b2 : b0;
                wyr[1] = r2 ? b3 : b1;
                wyr[2] = r2 ? b0 : b2;
                wyr[3] = r2 ? b1 : b3;
#pragma unroll
                for (int j = 0; j < P; ++j) row[j] = sm + off + (((uint32_t)j + r) & 3u) * EZ;
            }
#pragma unroll
            for (int jx = 0; jx < P; ++jx) {
#pragma unroll
                for (int jy = 0; jy < P; ++jy) {
                    const float wxy = wx[jx] * wyr[jy];
                    uint32_t* s = row[jy] + jx * EY * EZ;
#if TILD_SROT_FMUL2
                    {   // two packed multiplies (FMUL2, round to nearest, denormals kept) instead of four FMUL
                        const float2 v01 = fmul2_bcast(make_float2(wz[0], wz[1]), wxy), v23 = fmul2_bcast(make_float2(wz[2], wz[3]), wxy);
                        atomicAdd(s + 0, __float_as_uint(v01.x));
                        atomicAdd(s + 1, __float_as_uint(v01.y));
                        atomicAdd(s + 2, __float_as_uint(v23.x));
                        atomicAdd(s + 3, __float_as_uint(v23.y));
                    }
#else
#pragma unroll
                    for (int jz = 0; jz < P; ++jz) atomicAdd(s + jz, __float_as_uint(__fmul_rn(wxy, wz[jz])));
#endif
                }
            }
            ++n_tile;
        }
        {   // the queued drifted particles, one per thread (their fp32 reductions resolve in L2), taken by the LAST warps:
            // warp 0 always has the most rounds (k = wid, wid + SW, ...), the last ones the fewest
            const uint32_t nd = min(nq[par], (uint32_t)SDCAP);           // stable since the barrier after phase A
            const uint32_t td = (uint32_t)(ST - 1) - threadIdx.x;
            if (td < nd) spread_particle_global(m, X4[(size_t)c0 + dq[td]], grid);
        }
        __syncthreads();                             // the rounds are done: the lists are free, the image is complete so far
    }

    // flush: consecutive threads take consecutive z of a row so that the global reductions are coalesced along z
    unsigned long long tile_sum = 0;
    constexpr int RPP = ST / EZ;                     // rows per pass
    const int lz = threadIdx.x % EZ, r0 = threadIdx.x / EZ;
    const int gz = wrap_idx(o[2] + lz, m.N[2]);
    // A node can only wrap past 2^32 if >= 2^9 / (largest single-node weight) particles sit on it; the largest weight of
    // the cubic spline is (23/48)^3.  Tiles with fewer particles skip the check and the sum that feeds it.
    const bool check = p_hi - p_lo > 4653u;          // uniform across the block
    // 16-byte rows (Nz % 4 == 0: the image starts on a 16-byte boundary of the mesh rows, TileParams::sh, and every aligned
    // float4 of a row wraps as a whole): one vector reduction (red.global.add.v4.f32, REDG.E.ADD.F32x4) per four nodes
    const bool vec4 = !TILD_SROT_SCALAR_FLUSH && m.N[2] % 4 == 0 && (reinterpret_cast<uintptr_t>(grid) & 15) == 0 && (m.M % 4) == 0;
    auto flush = [&](auto sum, const float sc) {
        if (vec4) {
            constexpr int CPR = EZ / 4, RPP4 = ST / CPR;
            const int c4 = threadIdx.x % CPR, rr = threadIdx.x / CPR;
            if (rr >= RPP4) return;
            const int gz4 = wrap_idx(o[2] + 4 * c4, m.N[2]);
            for (int spl = 0; spl < nsp; ++spl) {
                float* gsp = grid + (size_t)(sp0 + spl) * m.M + gz4;
                const uint4* simg = reinterpret_cast<const uint4*>(sm + spl * E3) + c4;
                for (int q = rr; q < SEX * EY; q += RPP4) {
                    const uint4 u = simg[q * CPR];
                    if (u.x | u.y | u.z | u.w) {
                        if (decltype(sum)::value) tile_sum += (unsigned long long)u.x + u.y + u.z + u.w;
                        asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(gsp + rowoff[q]), "f"((float)u.x * sc),
                                     "f"((float)u.y * sc), "f"((float)u.z * sc), "f"((float)u.w * sc)
                                     : "memory");
                    }
                }
            }
            return;
        }
        if (r0 >= RPP) return;
        for (int spl = 0; spl < nsp; ++spl) {
            float* gsp = grid + (size_t)(sp0 + spl) * m.M + gz;
            const uint32_t* simg = sm + spl * E3 + lz;
            for (int q = r0; q < SEX * EY; q += RPP) {
                const uint32_t u = simg[q * EZ];
                if (u) {
                    if (decltype(sum)::value) tile_sum += u;
                    atomicAdd(gsp + rowoff[q], (float)u * sc);
                }
            }
        }
    };
#ifdef TILD_SROT_BULK_FLUSH
    // Bulk flush (measured, not the default): the image is converted to fp32 in place and every row goes to the mesh as one
    // (two across the periodic boundary in z) cp.reduce.async.bulk -- an fp32 add of 160 contiguous bytes done by the copy
    // engine in L2 -- instead of one RED per node issued by the SM.  Needs 16-byte rows: Nz % 4 == 0 (the image then starts
    // on a 16-byte boundary of the mesh rows, TileParams::sh) and an aligned grid.  C4: spread 0.2416 ms against 0.2382 ms for
    // the RED loop below, and 0.1887 ms with no flush at all: the flush is bound by the fp32 adds in L2 (137 M per step) and
    // the read-modify-write of the grid lines, not by who issues them (profiles/r2_variants.md).
    if (m.N[2] % 4 == 0 && EZ <= m.N[2] && (reinterpret_cast<uintptr_t>(grid) & 15) == 0) {   // uniform
        const int n4 = nsp * E3 / 4;
        uint4* v4 = reinterpret_cast<uint4*>(sm);
        for (int k = threadIdx.x; k < n4; k += ST) {
            const uint4 u = v4[k];
            if (check) tile_sum += (unsigned long long)u.x + u.y + u.z + u.w;
            reinterpret_cast<float4*>(sm)[k] = make_float4((float)u.x * FIX_INV, (float)u.y * FIX_INV, (float)u.z * FIX_INV, (float)u.w * FIX_INV);
        }
        const int gz0 = wrap_idx(o[2], m.N[2]);
        const int len1 = min(EZ, m.N[2] - gz0);      // floats before the periodic boundary; a multiple of 4
        auto bulk_rows = [&]() {
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // the image was written through the generic proxy
            __syncthreads();
            for (int r = threadIdx.x; r < nsp * SEX * EY; r += ST) {
                const int spl = r / (SEX * EY), q = r - spl * (SEX * EY);
                if (q % EY >= E[1]) continue;        // rows of the template image this tile shape does not use
                float* g = grid + (size_t)(sp0 + spl) * m.M + rowoff[q];
                const unsigned src = (unsigned)__cvta_generic_to_shared(sm + spl * E3 + q * EZ);
                asm volatile("cp.reduce.async.bulk.global.shared::cta.bulk_group.add.f32 [%0], [%1], %2;" ::"l"(g + gz0), "r"(src), "r"(4 * len1)
                             : "memory");
                if (len1 < EZ)
                    asm volatile("cp.reduce.async.bulk.global.shared::cta.bulk_group.add.f32 [%0], [%1], %2;" ::"l"(g), "r"(src + 4u * len1),
                                 "r"(4 * (EZ - len1))
                                 : "memory");
            }
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
            asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");   // the engine has read the image
        };
        bulk_rows();
        if (!check) return;
        const unsigned long long total = block_sum_u64(tile_sum, red);
        const unsigned long long cntp = block_sum_u64((unsigned long long)n_tile, red);
        const unsigned long long expect = cntp << FIX_BITS, slack = 64ull * cntp + 64ull;
        if (total + slack >= expect && total <= expect + slack) return;   // uniform across the block
        __syncthreads();
        for (int k = threadIdx.x; k < nsp * E3; k += ST) sm[k] ^= 0x80000000u;   // undo the wrapped tile: add the negated image
        bulk_rows();
    } else
#endif
    {
        if (!check) {
            flush(std::false_type(), FIX_INV);
            return;
        }
        flush(std::true_type(), FIX_INV);
        const unsigned long long total = block_sum_u64(tile_sum, red);
        const unsigned long long cntp = block_sum_u64((unsigned long long)n_tile, red);
        const unsigned long long expect = cntp << FIX_BITS, slack = 64ull * cntp + 64ull;
        if (total + slack >= expect && total <= expect + slack) return;   // uniform across the block
        flush(std::false_type(), -FIX_INV);              // undo the wrapped tile
    }
    // a node wrapped past 2^32 (>= 512 particles' worth on one node): redo this tile with fp32 global atomics
    for (uint32_t i = p_lo + threadIdx.x; i < p_hi; i += ST) {
        const float4 p = X4[i];
        const float pos[3] = {p.x, p.y, p.z};
        bool inside = true;
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            int cell, b;
            float t;
            index_1d<P>(pos[a], m.inv_h[a], cell, b, t);
            const int d = wrap_near(b - o[a], m.N[a]);
            inside = inside && ((unsigned)d + (unsigned)P <= (unsigned)E[a]);
        }
        if (inside) spread_particle_global(m, p, grid);   // the others went to the global grid in phase A already
    }
}

template <int EY, int EZ>
cudaError_t spread_rot_launch(const tild_ctx* c, int sp_group, size_t smem, const uint32_t* seg_base, const float4* X4, float* grid,
                              bool configure_only)
{
    auto kernel = spread_rot_kernel<EY, EZ>;
    if (configure_only) return tild_raise_smem_limit(reinterpret_cast<const void*>(kernel), smem);
    const dim3 g((unsigned)c->tile.nt[2], (unsigned)c->tile.nt[1], (unsigned)(c->tile.nt[0] * ((c->mesh.S + sp_group - 1) / sp_group)));
    kernel<<<g, ST, smem, c->stream>>>(c->mesh, c->tile, sp_group, seg_base, X4, grid);
    return cudaSuccess;
}

}  // namespace

// P = 4 with an image whose rows tile the banks (EZ = 24 or 40) and the default tile width in x
bool spread_rot_applies(const tild_ctx* c)
{
    const TileParams& t = c->tile;
    return t.enabled && c->mesh.P == 4 && t.E[0] == SEX && (t.EZ == 24 || t.EZ == 40) && (t.EY == 11 || t.EY == 19);
}

// species per CTA and dynamic shared memory of the instantiation this context uses
static void spread_rot_shape(const tild_ctx* c, int* sp_group, size_t* smem)
{
    const size_t per_species = (size_t)SEX * c->tile.EY * c->tile.EZ * sizeof(uint32_t);
    const size_t lists = (size_t)3 * SSLOTS * sizeof(uint32_t);
    int g = (int)((112 * 1024 - lists) / per_species);
    if (g < 1) g = 1;
    if (g > c->mesh.S) g = c->mesh.S;
    *sp_group = g;
    *smem = per_species * g + lists;
}

cudaError_t spread_rot_run(const tild_ctx* c, const uint32_t* seg_base, const float4* X4, float* grid, bool configure_only)
{
    int g;
    size_t smem;
    spread_rot_shape(c, &g, &smem);
    const int ey = c->tile.EY, ez = c->tile.EZ;
    if (ey == 19 && ez == 40) return spread_rot_launch<19, 40>(c, g, smem, seg_base, X4, grid, configure_only);
    if (ey == 19 && ez == 24) return spread_rot_launch<19, 24>(c, g, smem, seg_base, X4, grid, configure_only);
    if (ey == 11 && ez == 40) return spread_rot_launch<11, 40>(c, g, smem, seg_base, X4, grid, configure_only);
    return spread_rot_launch<11, 24>(c, g, smem, seg_base, X4, grid, configure_only);
}
