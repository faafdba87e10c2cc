// a6, cubic assignment (P = 4): mesh -> particle interpolation with the weights of the spread
// (Fig. 1) + bonds (Eq. 2) + integrator (L346-352) in one pass, second-generation
// tile kernel.  What bounds it is the shared-memory data pipe (128 B / clock / SM): every particle reads 3 x 64 words
// of the staged force field, so the kernel is organised around the number of LDS WAVEFRONTS and of L1 wavefronts
// spent on anything else (profiles/r2_interp_design.md):
//
//  * Rotation classes.  A round of 32 particles is free of bank conflicts when their first stencil nodes fall into
//    32 different banks ("class" = word offset mod 32, tild_interp.cu).  With 32 classes of ~32 particles the class
//    counts differ by +-35 %, which wasted 27 % of the wavefronts.  Here EZ = 8 mod 32 (or 24), so the P = 4 rows
//    (jy = 0..3) of a stencil start 0, 8, 16, 24 banks apart: traversing the rows in the rotated order (jy + r) mod 4
//    turns a particle of class c into one of class c + 8r.  Every particle therefore fits any of the 4 lanes
//    g, g+8, g+16, g+24 (g = c mod 8); the 4 lanes of a group are filled round-robin and only the 8 group totals
//    (~128 +- 8 %) remain unbalanced.  No overflow lists, no mixed rounds.
//  * The list entry carries what a round needs (three stencil offsets t as 25-bit fixed point -- t is a multiple of
//    2^-24 for all but the first half cell of an axis -- image offset, rotation) in 12 bytes of shared memory; the
//    same 12 bytes return the interpolated force to the thread that binned the particle.
//  * Bonds, Philox, integrator and all global traffic of a particle run in SLOT order by the thread that binned it:
//    coalesced 16-byte loads and stores instead of accesses scattered in class order (a third of the L1 wavefronts
//    of the first-generation kernel).
//  * The four z nodes of a row are accumulated with the (w_x w_y) weight and the z weights are applied once at the end
//    (192 + 12 FMAs per particle instead of 240).  The packed FFMA2 form of the same sums (96 instructions) measured
//    7 % slower (0.695 vs 0.650 ms) and is kept behind TILD_USE_FFMA2.
//  * Software pipeline over the chunks of a tile: the next chunk's positions and partners are loaded while this
//    chunk's tail computes; this chunk's velocity state and partner positions are loaded before its rounds.
#include <cuda.h>   // CUtensorMap (types only: the encoder is fetched with cudaGetDriverEntryPoint, libcuda is not linked)

#include "tild_particle.cuh"

namespace {

// TILD_ROT_PROFILE (experiments only): thread 0 of every CTA accumulates clock64() deltas per phase into F4 (unused by MODE 2)
#ifdef TILD_ROT_PROFILE
#define PROF_DECL long long pt_[8] = {0, 0, 0, 0, 0, 0, 0, 0}, pc_ = clock64();
#define PROF_MARK(k) do { if (threadIdx.x == 0) { const long long n_ = clock64(); pt_[k] += n_ - pc_; pc_ = n_; } } while (0)
#define PROF_DUMP() do { if (threadIdx.x == 0 && MODE == 2) { F4[2 * tile] = make_float4((float)pt_[0], (float)pt_[1], (float)pt_[2], (float)pt_[3]); F4[2 * tile + 1] = make_float4((float)pt_[4], (float)pt_[5], (float)pt_[6], (float)pt_[7]); } } while (0)
#else
#define PROF_DECL
#define PROF_MARK(k)
#define PROF_DUMP()
#endif

#ifndef TILD_ROT_ABL
#define TILD_ROT_ABL 0   // experiments only: 1 no staging, 2 no rounds, 4 no partner loads, 8 no tail
#endif
// 256 threads x 2 CTAs per SM (128 registers, no spills: with the whole L1 carved out as shared memory a spill is an L2
// round trip), 512 particles binned at a time (2 per thread).  Measured alternatives: profiles/r2_interp_variants.md.
#ifndef TILD_ROT_THREADS
#define TILD_ROT_THREADS 256
#define TILD_ROT_CTAS 2
#define TILD_ROT_CHUNK 512
#define TILD_ROT_KCAP 22
#endif
constexpr int RT = TILD_ROT_THREADS;    // threads per CTA
constexpr int RW = RT / 32;
constexpr int RCHUNK = TILD_ROT_CHUNK;  // particles binned at a time
constexpr int RPT = (RCHUNK + RT - 1) / RT;   // particles per thread and chunk
constexpr int RKCAP = TILD_ROT_KCAP;    // rounds of list space (mean RCHUNK / 32 for a full chunk)
constexpr int RSLOTS = RKCAP * 32;
constexpr int RDCAP = 112;              // drifted particles per tile handed over with one global atomic
constexpr int REX = 11;                 // image edge in x: 8 cells + halo 3

__device__ __forceinline__ void cp_async_f32(float* smem_dst, const float* gsrc)
{
    const unsigned sa = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;\n" ::"r"(sa), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_16(float* smem_dst, const float* gsrc)
{
    const unsigned sa = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(sa), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;\n" ::: "memory"); }

// ---- TMA (cp.async.bulk.tensor) staging of a tile image, for tiles whose image does not cross the periodic boundary ------
__device__ __forceinline__ void mbar_init(uint64_t* bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, unsigned parity)
{
    const unsigned a = (unsigned)__cvta_generic_to_shared(bar);
    unsigned done = 0;
    while (!done)
        asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}" : "=r"(done) : "r"(a), "r"(parity) : "memory");
}
// one box {EZ, EY, REX, 1} of the 4-D field [3S][Nx][Ny][Nz] -> dense image of one component
__device__ __forceinline__ void tma_load_box(float* smem_dst, const CUtensorMap* map, int z, int y, int x, int f, uint64_t* bar)
{
    asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];" ::
                     "r"((unsigned)__cvta_generic_to_shared(smem_dst)), "l"(map), "r"(z), "r"(y), "r"(x), "r"(f),
                 "r"((unsigned)__cvta_generic_to_shared(bar))
                 : "memory");
}

#ifdef TILD_ROT_DRIFT_IN_CTA
// one drifted particle: global gather of its stencil + the tail (experiment, see the end of the kernel)
template <int MODE>
__device__ __noinline__ void drifted_particle(const MeshParams& m, const StepParams& s, uint64_t step_next, size_t slot,
                                              const float* __restrict__ ffield, const float4* __restrict__ X4,
                                              const float4* __restrict__ W4, const int32_t* __restrict__ B, float4* __restrict__ X4o,
                                              float4* __restrict__ W4o, float4* __restrict__ F4)
{
    const float4 p = X4[slot];
    int b[3];
    float w[3][4];
    index_weights<4>(m, p, b, w);
    const bool vec = (m.N[2] % 4 == 0) && ((reinterpret_cast<uintptr_t>(ffield) & 15) == 0);
    const float3 F = vec ? interp_global<4, true>(m, ffield, b, w, __float_as_int(p.w)) : interp_global<4, false>(m, ffield, b, w, __float_as_int(p.w));
    finish_particle<MODE>(m, s, step_next, slot, p, F, X4, W4, B, X4o, W4o, F4);
}
#endif

// Dynamic shared memory: (128-byte aligned) image float[3][CSP] of one species, CSP = REX EY EZ rounded up to 32 words so that
// every component starts on a 128-byte boundary (TMA destination) | ent u32[3][RSLOTS].
// FAST (MODE 2 only): the plain model of BASELINE configs -- two bond slots, no rest length, no angle potentials, three
// dimensions, an inertial integrator.  The fields that select the other paths become compile-time constants, which removes
// their (never taken, but scheduling-relevant) branches from the hot kernel.
template <int EY, int EZ, int MODE, bool FAST>
__global__ void __launch_bounds__(RT, TILD_ROT_CTAS) interp_rot_kernel(MeshParams m, TileParams tp, StepParams s_in, const uint64_t* __restrict__ step_ptr,
                                                          const uint32_t* __restrict__ seg_base, const float* __restrict__ ffield,
                                                          const float4* __restrict__ X4, const float4* __restrict__ W4,
                                                          const int32_t* __restrict__ B, float4* __restrict__ X4o,
                                                          float4* __restrict__ W4o, float4* __restrict__ F4,
                                                          uint32_t* __restrict__ drift_list, uint32_t* __restrict__ drift_count,
                                                          const __grid_constant__ CUtensorMap fmap, int use_tma,
                                                          float4* __restrict__ zgrid, size_t zcount4, size_t zper)
{
    constexpr int P = 4, CS = (REX * EY * EZ + 31) / 32 * 32;
    // grid (nt_z, nt_y, nt_x): the tile coordinates are the block indices (no integer divisions), launch order = tile order
    const int tz = blockIdx.x, ty = blockIdx.y, tx = blockIdx.z;
    const int tile = (tx * tp.nt[1] + ty) * tp.nt[2] + tz;
    // The density grid of the next step, cleared here (an equal share per CTA) instead of by a memset in front of the spread:
    // this kernel is bound by the shared-memory pipe and leaves most of the HBM bandwidth unused.
    if (MODE == 2 && zgrid) {
        const size_t z0 = (size_t)tile * zper, z1 = min(z0 + zper, zcount4);   // zper = ceil(zcount4 / tiles), from the host
        for (size_t i = z0 + threadIdx.x; i < z1; i += RT) zgrid[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    static_assert(EZ % 32 == 8 || EZ % 32 == 24, "row rotation needs the P rows of a stencil to tile the 32 banks");
    static_assert(!FAST || MODE == 2, "FAST is a specialisation of the fused step");
    StepParams s = s_in;
    fold_plain_model<FAST>(s);
    extern __shared__ __align__(16) float fs_raw[];
    // 128-byte alignment for the TMA boxes, as an offset in the shared window: a round trip through uintptr_t would lose the
    // address space and turn every stencil LDS into a generic LD with 64-bit address arithmetic
    float* fs = fs_raw + (((128u - ((unsigned)__cvta_generic_to_shared(fs_raw) & 127u)) & 127u) >> 2);
    __shared__ int goff_x[16], goff_y[32];
    __shared__ uint32_t gcnt[8], ndrift, drift_base, dl[RDCAP];
    __shared__ __align__(8) uint64_t mbar;
    uint32_t* ent = reinterpret_cast<uint32_t*>(fs + 3 * CS);
    const uint64_t step_next = *step_ptr + 1;   // the step being produced (device-side counter: graph replays see it move)
    const int o[3] = {tx * tp.T[0] - tp.lo, ty * tp.T[1] - tp.lo, tz * tp.T[2] - tp.lo - tp.sh};
    const int E[3] = {REX, tp.E[1], EZ};
    const size_t seg0 = (size_t)tile * m.S;
    if (seg_base[seg0] == seg_base[seg0 + m.S]) return;   // empty tile (uniform)
    if (threadIdx.x < REX) goff_x[threadIdx.x] = wrap_idx(o[0] + threadIdx.x, m.N[0]);
    else if (threadIdx.x >= 32 && threadIdx.x < 32 + EY) goff_y[threadIdx.x - 32] = wrap_idx(o[1] + threadIdx.x - 32, m.N[1]);
    if (threadIdx.x >= 64 && threadIdx.x < 72) gcnt[threadIdx.x - 64] = 0u;
    if (threadIdx.x == 72) ndrift = 0u;
    // TMA staging when the whole image lies inside the mesh (61 % of the tiles at 256^3): one box per component, issued by
    // one thread, completion on an mbarrier; the other tiles wrap per row with cp.async below
    const bool tma_tile = use_tma && o[0] >= 0 && o[0] + REX <= m.N[0] && o[1] >= 0 && o[1] + EY <= m.N[1] && o[2] >= 0 && o[2] + EZ <= m.N[2];
    unsigned tma_parity = 0;
    if (tma_tile && threadIdx.x == 0) {
        mbar_init(&mbar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const bool vec16 = (m.N[2] % 4 == 0) && ((reinterpret_cast<uintptr_t>(ffield) & 15) == 0);

    auto stage = [&](int sp) {   // three components of species sp -> image (periodic wrap per row); asynchronous
        if (TILD_ROT_ABL & 1) return;
        if (tma_tile) {
            if (threadIdx.x == 0) {
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // the image was read through the generic proxy
                mbar_expect_tx(&mbar, 3u * REX * EY * EZ * (unsigned)sizeof(float));
#pragma unroll
                for (int comp = 0; comp < 3; ++comp) tma_load_box(fs + comp * CS, &fmap, o[2], o[1], o[0], sp * 3 + comp, &mbar);
            }
            return;
        }
        const float* fsp = ffield + (size_t)sp * 3 * m.FM;
        if (vec16) {
            // 16-byte copies: the image starts on a 16-byte boundary of the mesh rows (tp.sh) and Nz % 4 == 0,
            // so every aligned float4 of a row stays inside the row and wraps as a whole
            constexpr int CPR = EZ / 4, RPP = RT / CPR;
            const int chunk = threadIdx.x % CPR;
            const int gz = wrap_idx(o[2] + 4 * chunk, m.N[2]);
            if (threadIdx.x < RPP * CPR)
                for (int q = threadIdx.x / CPR; q < REX * EY; q += RPP) {
                    const int lx = q / EY, ly = q - lx * EY;
                    if (ly >= E[1]) continue;
                    const float* src = fsp + ((size_t)goff_x[lx] * m.FN[0] + goff_y[ly]) * m.FN[1] + gz;
                    float* dst = fs + q * EZ + 4 * chunk;
#pragma unroll
                    for (int comp = 0; comp < 3; ++comp) cp_async_16(dst + comp * CS, src + (size_t)comp * m.FM);
                }
        } else {
            constexpr int RPP = RT / EZ;
            const int lz = threadIdx.x % EZ;
            const int gz = wrap_idx(o[2] + lz, m.N[2]);
            if (threadIdx.x < RPP * EZ)
                for (int q = threadIdx.x / EZ; q < REX * EY; q += RPP) {
                    const int lx = q / EY, ly = q - lx * EY;
                    if (ly >= E[1]) continue;
                    const float* src = fsp + ((size_t)goff_x[lx] * m.FN[0] + goff_y[ly]) * m.FN[1] + gz;
                    float* dst = fs + q * EZ + lz;
#pragma unroll
                    for (int comp = 0; comp < 3; ++comp) cp_async_f32(dst + comp * CS, src + (size_t)comp * m.FM);
                }
        }
        cp_async_commit();
    };

    // work items: (species, chunk) in order; the image of a species is staged when its first chunk starts.
    // Software pipeline over the work items (the shared-memory carve-out leaves no L1, every global load is an L2 or DRAM
    // round trip): positions and bond partners of the NEXT chunk are loaded while the tail of this one computes; the
    // velocity state and the partners' positions of THIS chunk are loaded before its rounds and used after them.
    int sp = 0;
    while (sp < m.S && seg_base[seg0 + sp] == seg_base[seg0 + sp + 1]) ++sp;
    uint32_t p_lo = seg_base[seg0 + sp], p_hi = seg_base[seg0 + sp + 1];
    uint32_t per = (p_hi - p_lo + RCHUNK - 1) / RCHUNK;           // chunks of this segment
    per = ((p_hi - p_lo + per - 1) / per + 31u) & ~31u;           // equal chunks, whole rounds
    uint32_t c0 = p_lo;
    const bool two_bonds = MODE >= 1 && s.max_bonds == 2, one_bond = MODE >= 1 && s.max_bonds == 1;
    auto load_chunk = [&](uint32_t base, int cnt, float4 (&px)[RPT], int2 (&pb)[RPT]) {
#pragma unroll
        for (int j = 0; j < RPT; ++j) {
            const int i = threadIdx.x + j * RT;
            pb[j] = make_int2(-1, -1);
            if (i >= cnt) continue;
            px[j] = X4[(size_t)base + i];
            if (two_bonds) pb[j] = *reinterpret_cast<const int2*>(B + 2 * ((size_t)base + i));
            else if (one_bond) pb[j].x = B[(size_t)base + i];
        }
    };
    PROF_DECL
    float4 pa[RPT];
    int2 ba[RPT];
    load_chunk(c0, (int)min(per, p_hi - c0), pa, ba);
    __syncthreads();                                              // goff_*, gcnt, mbarrier visible
    bool staged = true;                                           // an image is on its way (uniform)
    stage(sp);
    PROF_MARK(0);                                                 // 0: prologue + staging issue
    while (true) {
        const int nchunk = (int)min(per, p_hi - c0);
        // ---- phase A: bin by rotation group; the thread keeps the list slots of its particles ----------------------
        int myslot[RPT];
#pragma unroll
        for (int j = 0; j < RPT; ++j) {
            const int i = threadIdx.x + j * RT;
            myslot[j] = -1;
            if (i >= nchunk) continue;
            const float4 p = pa[j];
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
            uint32_t k = RKCAP, pos4 = 0, off = 0;
            if (inside) {
                off = (uint32_t)((d[0] * EY + d[1]) * EZ + d[2]);
                pos4 = atomicAdd(&gcnt[off & 7u], 1u);
                k = pos4 >> 2;
            }
            if (k < RKCAP) {
                const uint32_t ln = (off & 7u) + 8u * (pos4 & 3u);    // lane that will take it
                // rows traversed as (jy + r) mod 4: moves the particle from class off to class off + r RB (mod 32), RB = EZ mod 32
                const uint32_t r = ((EZ % 32 == 8 ? ln - off : off - ln) >> 3) & 3u;
                const uint32_t slot = k * 32u + ln;
                const int q0 = __float2int_rn(t[0] * 16777216.0f), q1 = __float2int_rn(t[1] * 16777216.0f),
                          q2 = __float2int_rn(t[2] * 16777216.0f);
                ent[slot] = ((uint32_t)q0 & 0x1FFFFFFu) | (off << 25);
                ent[RSLOTS + slot] = ((uint32_t)q1 & 0x1FFFFFFu) | ((off >> 7) << 25);
                ent[2 * RSLOTS + slot] = ((uint32_t)q2 & 0x1FFFFFFu) | (r << 25);
                myslot[j] = (int)slot;
            } else {
                // left the tile's image since the last re-sort (or no list space): handed to interp_drift_kernel through
                // a per-tile list (one global atomic per tile at the end); beyond its capacity, one atomic per particle
                myslot[j] = -2;
                const uint32_t dj = atomicAdd(&ndrift, 1u);
                if (dj < (uint32_t)RDCAP) dl[dj] = c0 + (uint32_t)i;
                else drift_list[atomicAdd(drift_count, 1u)] = c0 + (uint32_t)i;
            }
        }
        // loads the tail of this chunk needs, in flight during the rounds: velocity state, partners' positions
        float4 wj[RPT], q0[RPT], q1[RPT];
#pragma unroll
        for (int j = 0; j < RPT; ++j) {
            if (myslot[j] < 0) continue;
            if (MODE == 2) wj[j] = W4[(size_t)c0 + threadIdx.x + j * RT];
            // a missing partner reads the particle itself: zero separation, zero bond force, no branch in the tail
            q0[j] = X4[(ba[j].x >= 0 && !(TILD_ROT_ABL & 4)) ? (size_t)ba[j].x : (size_t)c0 + threadIdx.x + j * RT];
            q1[j] = X4[(ba[j].y >= 0 && !(TILD_ROT_ABL & 4)) ? (size_t)ba[j].y : (size_t)c0 + threadIdx.x + j * RT];
        }
        {   // L2 prefetch of the next chunk's lines (positions, partners, velocity state)
            const size_t nx = (size_t)c0 + nchunk + 8 * (size_t)threadIdx.x;
            if (threadIdx.x < RCHUNK / 8 && nx < (size_t)m.n) {
                asm volatile("prefetch.global.L2 [%0];" ::"l"(X4 + nx));
                if (MODE == 2) asm volatile("prefetch.global.L2 [%0];" ::"l"(W4 + nx));
            }
            const size_t nb = (size_t)c0 + nchunk + 16 * (size_t)threadIdx.x;
            if (two_bonds && threadIdx.x < RCHUNK / 16 && nb < (size_t)m.n) asm volatile("prefetch.global.L2 [%0];" ::"l"(B + 2 * nb));
        }
        PROF_MARK(1);                                                 // 1: binning
        cp_async_wait_all();
        if (tma_tile && staged) {                                     // the boxes of this species have landed
            mbar_wait(&mbar, tma_parity);
            tma_parity ^= 1u;
        }
        staged = false;
        PROF_MARK(2);                                                 // 2: wait for the image
        __syncthreads();
        PROF_MARK(3);                                                 // 3: barrier after binning
        // ---- rounds: lane l takes the k-th quadruple of group l & 7 --------------------------------------------------
        {
            const uint32_t mine = min(gcnt[lane & 7], (uint32_t)(4 * RKCAP));
            uint32_t rounds = mine;
#pragma unroll
            for (int dlt = 4; dlt > 0; dlt >>= 1) rounds = max(rounds, __shfl_xor_sync(0xffffffffu, rounds, dlt));
            rounds = (rounds + 3u) >> 2;
            if (!(TILD_ROT_ABL & 2))
            for (uint32_t k = wid; k < rounds; k += RW) {
                if (4u * k + (uint32_t)(lane >> 3) >= mine) continue;
                const uint32_t slot = k * 32u + lane;
                const uint32_t e0 = ent[slot], e1 = ent[RSLOTS + slot], e2 = ent[2 * RSLOTS + slot];
                const float tx_ = (float)((int)(e0 << 7) >> 7) * (1.0f / 16777216.0f);
                const float ty_ = (float)((int)(e1 << 7) >> 7) * (1.0f / 16777216.0f);
                const float tz_ = (float)((int)(e2 << 7) >> 7) * (1.0f / 16777216.0f);
                const uint32_t off = (e0 >> 25) | ((e1 >> 25) << 7), r = (e2 >> 25) & 3u;
                float wx[P], wy[P], wz[P];
                weights_1d<P>(tx_, wx);
                weights_1d<P>(ty_, wy);
                weights_1d<P>(tz_, wz);
                // rotated row order: row j of the traversal is stencil row (j + r) & 3
                const float* row[P];
                float wyr[P];
                {
                    const bool r1 = r & 1u, r2 = r & 2u;
                    const float b0 = r1 ? wy[1] : wy[0], b1 = r1 ? wy[2] : wy[1], b2 = r1 ? wy[3] : wy[2], b3 = r1 ? wy[0] : wy[3];
                    wyr[0] = r2 ? b2 : b0;
                    wyr[1] = r2 ? b3 : b1;
                    wyr[2] = r2 ? b0 : b2;
                    wyr[3] = r2 ? b1 : b3;
#pragma unroll
                    for (int j = 0; j < P; ++j) row[j] = fs + off + (((uint32_t)j + r) & 3u) * EZ;
                }
                float2 a01[3], a23[3];
#pragma unroll
                for (int c = 0; c < 3; ++c) a01[c] = a23[c] = make_float2(0.f, 0.f);
#pragma unroll
                for (int jx = 0; jx < P; ++jx) {
#pragma unroll
                    for (int jy = 0; jy < P; ++jy) {
                        const float wxy = wx[jx] * wyr[jy];
                        const float* f = row[jy] + jx * EY * EZ;
#pragma unroll
                        for (int c = 0; c < 3; ++c) {
                            a01[c] = ffma2_bcast(make_float2(f[c * CS], f[c * CS + 1]), wxy, a01[c]);
                            a23[c] = ffma2_bcast(make_float2(f[c * CS + 2], f[c * CS + 3]), wxy, a23[c]);
                        }
                    }
                }
                float F[3];
#pragma unroll
                for (int c = 0; c < 3; ++c) F[c] = (wz[0] * a01[c].x + wz[1] * a01[c].y) + (wz[2] * a23[c].x + wz[3] * a23[c].y);
                ent[slot] = __float_as_uint(F[0]);
                ent[RSLOTS + slot] = __float_as_uint(F[1]);
                ent[2 * RSLOTS + slot] = __float_as_uint(F[2]);
            }
        }
        PROF_MARK(4);                                                 // 4: rounds
        __syncthreads();
        PROF_MARK(5);                                                 // 5: barrier after the rounds
        // the next work item; its image (if it is a new species) is staged and its particles are loaded while the tail
        // below computes
        const uint32_t c0_done = c0;
        bool more = true;
        c0 += (uint32_t)nchunk;
        if (c0 >= p_hi) {
            do ++sp; while (sp < m.S && seg_base[seg0 + sp] == seg_base[seg0 + sp + 1]);
            if (sp < m.S) {
                p_lo = seg_base[seg0 + sp];
                p_hi = seg_base[seg0 + sp + 1];
                per = (p_hi - p_lo + RCHUNK - 1) / RCHUNK;
                per = ((p_hi - p_lo + per - 1) / per + 31u) & ~31u;
                c0 = p_lo;
                staged = true;
                stage(sp);
            } else {
                more = false;
            }
        }
        float4 pn[RPT];
        int2 bn[RPT];
        if (more) load_chunk(c0, (int)min(per, p_hi - c0), pn, bn);
        if (threadIdx.x < 8) gcnt[threadIdx.x] = 0u;   // the rounds are done with the counts
        // ---- tail in slot order: bonds, noise, integrator; coalesced global traffic ---------------------------------
        if (!(TILD_ROT_ABL & 8)) {
#pragma unroll
            for (int j = 0; j < RPT; ++j) {
                const size_t slot = (size_t)c0_done + threadIdx.x + j * RT;
                if (myslot[j] < 0) continue;
                float3 F = make_float3(__uint_as_float(ent[myslot[j]]), __uint_as_float(ent[RSLOTS + myslot[j]]),
                                       __uint_as_float(ent[2 * RSLOTS + myslot[j]]));
                const float4 p = pa[j];
                if (MODE >= 1) {
                    if (s.max_bonds <= 2) {
                        bond_term(m, s, p, q0[j], F);
                        bond_term(m, s, p, q1[j], F);
                        if (s.lambda_wlc != 0.0f || s.k_theta != 0.0f) angle_force_slots(m, s, X4, B, slot, p, F);
                    } else {
                        const float3 fb = bond_force_slots(m, s, X4, B, slot, p);
                        F.x += fb.x;
                        F.y += fb.y;
                        F.z += fb.z;
                    }
                }
                finish_update<MODE>(m, s, step_next, slot, p, F, MODE == 2 ? wj[j] : make_float4(0.f, 0.f, 0.f, 0.f), X4o, W4o, F4);
            }
        }
        PROF_MARK(6);                                                 // 6: staging issue + tail
        if (!more) break;
        __syncthreads();                                              // the tail has read its forces: the lists are free
#pragma unroll
        for (int j = 0; j < RPT; ++j) {
            pa[j] = pn[j];
            ba[j] = bn[j];
        }
    }
    PROF_DUMP();
    __syncthreads();
    const uint32_t nd = min(ndrift, (uint32_t)RDCAP);                  // uniform
    if (nd == 0) return;
#ifndef TILD_ROT_DRIFT_IN_CTA
    // handed to interp_drift_kernel.  (Doing them here, one per thread from the global field while it is L2-hot, measured
    // 0.837 instead of 0.582 ms: the gather's latency sits at the end of every CTA and holds its SM slot.)
    if (threadIdx.x == 0) drift_base = atomicAdd(drift_count, nd);
    __syncthreads();
    if (threadIdx.x < nd) drift_list[drift_base + threadIdx.x] = dl[threadIdx.x];
#else
    if (threadIdx.x < nd) drifted_particle<MODE>(m, s, step_next, dl[threadIdx.x], ffield, X4, W4, B, X4o, W4o, F4);
#endif
}

template <int EY, int EZ, int MODE, bool FAST>
cudaError_t rot_launch(const InterpArgs& a, cudaStream_t st, size_t smem, bool configure_only)
{
    auto kernel = interp_rot_kernel<EY, EZ, MODE, FAST>;
    if (configure_only) return tild_raise_smem_limit(reinterpret_cast<const void*>(kernel), smem);
    static const CUtensorMap no_map{};
    const bool tma = a.use_tma && a.tp.E[1] == EY;     // the box of the tensor map is the template image
    const CUtensorMap* map = tma ? static_cast<const CUtensorMap*>(a.fmap) : &no_map;
    const dim3 g((unsigned)a.tp.nt[2], (unsigned)a.tp.nt[1], (unsigned)a.tp.nt[0]);
    kernel<<<g, RT, smem, st>>>(a.m, a.tp, a.s, a.step_ptr, a.seg_base, a.ffield, a.X4, a.W4, a.B, a.X4o, a.W4o, a.F4,
                                a.drift_list, a.drift_count, *map, tma ? 1 : 0, MODE == 2 ? a.zgrid : nullptr, a.zcount4,
                                (a.zcount4 + (size_t)a.tp.ntiles - 1) / (size_t)a.tp.ntiles);
    return cudaSuccess;
}
template <int EY, int EZ>
cudaError_t rot_launch_m(const InterpArgs& a, int mode, cudaStream_t st, size_t smem, bool cfg)
{
    const bool fast = plain_model(a.s);
    cudaError_t e = cudaSuccess, e2;
    if (cfg || mode == 0) { e2 = rot_launch<EY, EZ, 0, false>(a, st, smem, cfg); if (e2 != cudaSuccess) e = e2; }
    if (cfg || mode == 1) { e2 = rot_launch<EY, EZ, 1, false>(a, st, smem, cfg); if (e2 != cudaSuccess) e = e2; }
    if (cfg || (mode == 2 && !fast)) { e2 = rot_launch<EY, EZ, 2, false>(a, st, smem, cfg); if (e2 != cudaSuccess) e = e2; }
    if (cfg || (mode == 2 && fast)) { e2 = rot_launch<EY, EZ, 2, true>(a, st, smem, cfg); if (e2 != cudaSuccess) e = e2; }
    return e;
}

}  // namespace

size_t interp_rot_smem(int ey, int ez)
{
    const size_t csp = ((size_t)REX * ey * ez + 31) / 32 * 32;      // component stride, 128-byte multiple
    return csp * 3 * sizeof(float) + (size_t)3 * RSLOTS * sizeof(uint32_t) + 128;   // + alignment slack
}

// Tensor map of the library's force field [3S][Nx][Ny][Nz] (float, z fastest) with the box of one component image.
// Returns false when TMA cannot be used (rows not 16-byte multiples, driver entry point missing): cp.async staging then.
bool interp_rot_make_tmap(tild_ctx* c)
{
    c->tma_ok = false;
    if (!interp_rot_applies(c) || c->mesh.N[2] % 4 != 0 || (c->prm.flags & TILD_FLAG_NO_TMA)) return false;
    typedef CUresult (*encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                  const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn || qres != cudaDriverEntryPointSuccess) {
        cudaGetLastError();
        return false;
    }
    const cuuint64_t dims[4] = {(cuuint64_t)c->mesh.N[2], (cuuint64_t)c->mesh.N[1], (cuuint64_t)c->mesh.N[0], (cuuint64_t)(3 * c->mesh.S)};
    const cuuint64_t strides[3] = {(cuuint64_t)c->mesh.N[2] * 4, (cuuint64_t)c->mesh.N[2] * c->mesh.N[1] * 4, (cuuint64_t)c->M * 4};
    const cuuint32_t box[4] = {(cuuint32_t)c->tile.EZ, (cuuint32_t)c->tile.EY, (cuuint32_t)REX, 1u};
    const cuuint32_t estr[4] = {1u, 1u, 1u, 1u};
    static_assert(sizeof(CUtensorMap) <= sizeof(c->fmap), "tensor map storage");
    const CUresult r = reinterpret_cast<encode_fn>(fn)(reinterpret_cast<CUtensorMap*>(c->fmap), CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, c->ffield, dims,
                                                       strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                                       CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    c->tma_ok = r == CUDA_SUCCESS;
    return c->tma_ok;
}

// P = 4 with an image whose rows tile the banks (EZ = 24 or 40) and the default tile width in x
bool interp_rot_applies(const tild_ctx* c)
{
    const TileParams& t = c->tile;
    return t.enabled && c->mesh.P == 4 && t.E[0] == REX && (t.EZ == 24 || t.EZ == 40) && (t.EY == 11 || t.EY == 19);
}

// configure_only: raise the shared-memory limit of the instantiation this context uses (all three modes)
cudaError_t interp_rot_run(const InterpArgs& a, int mode, cudaStream_t st, bool configure_only)
{
    const size_t smem = interp_rot_smem(a.tp.EY, a.tp.EZ);
    if (a.tp.EY == 19 && a.tp.EZ == 40) return rot_launch_m<19, 40>(a, mode, st, smem, configure_only);
    if (a.tp.EY == 19 && a.tp.EZ == 24) return rot_launch_m<19, 24>(a, mode, st, smem, configure_only);
    if (a.tp.EY == 11 && a.tp.EZ == 40) return rot_launch_m<11, 40>(a, mode, st, smem, configure_only);
    return rot_launch_m<11, 24>(a, mode, st, smem, configure_only);
}
