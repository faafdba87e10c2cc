// a6: mesh -> particle interpolation with the same weights (Fig. 1),
// harmonic bonds computed per particle without Newton's third law (Eq. 2) and the GJF Langevin
// update (L352; equations per DESIGN.md A11) fused into one pass over the particles.
//
// Hot kernel: one CTA per tile.  For each species present in the tile the three force-field components of the
// tile (+ stencil halo) are staged into shared memory with 16-byte cp.async row copies (periodic wrap applied per
// row).  While those copies are in flight the CTA bins the segment's particles by the bank of their first stencil
// node in the image ("class", see tild_spread.cu), then works in rounds of one particle per class: lane c takes
// the k-th particle of class c, so each of the 3 P^3 shared-memory loads of the stencil hits 32 different banks.
#include "tild_particle.cuh"

namespace {

constexpr int INTERP_THREADS = 384;
constexpr int INTERP_WARPS = INTERP_THREADS / 32;


// per-particle kernel over the slots [s0, s1)
template <int P, bool VEC, int MODE, bool FAST>
__global__ void __launch_bounds__(256, P == 1 ? (FAST ? 8 : 4) : 1) interp_slots_kernel(MeshParams m, StepParams s_in, const uint64_t* __restrict__ step_ptr, size_t s0, size_t s1,
                                                           const float* __restrict__ ffield, const float4* __restrict__ X4,
                                                           const float4* __restrict__ W4, const int32_t* __restrict__ B,
                                                           float4* __restrict__ X4o, float4* __restrict__ W4o,
                                                           float4* __restrict__ F4)
{
    StepParams s = s_in;
    fold_plain_model<FAST>(s);
    const uint64_t step_next = *step_ptr + 1;   // the step being produced (device-side counter: graph replays see it move)
    const size_t slot = s0 + (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (slot >= s1) return;
    const float4 p = X4[slot];
    const int type = __float_as_int(p.w);
    int b[3];
    float w[3][P];
    index_weights<P>(m, p, b, w);
    const float3 F = interp_global<P, VEC>(m, ffield, b, w, type);
    finish_particle<MODE>(m, s, step_next, slot, p, F, X4, W4, B, X4o, W4o, F4);
}

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

// Dynamic shared memory: image float[3][EX][EY][EZ] of one species | idx u16[KCAP][32] | ovf u16[CHUNK].
// FAST (MODE 2): the plain model (two bond slots, no rest length, no angles, 3-D, inertial integrator) with those facts
// folded in at compile time: no call sites of the generic bond / angle routines, hence no registers saved around them.
template <int P, int EY, int EZ, int MODE, bool FAST>
__global__ void __launch_bounds__(INTERP_THREADS, 2) interp_tile_kernel(MeshParams m, TileParams tp, StepParams s_in, const uint64_t* __restrict__ step_ptr,
                                                                     const uint32_t* __restrict__ seg_base,
                                                                     const float* __restrict__ ffield,
                                                                     const float4* __restrict__ X4, const float4* __restrict__ W4,
                                                                     const int32_t* __restrict__ B, float4* __restrict__ X4o,
                                                                     float4* __restrict__ W4o, float4* __restrict__ F4,
                                                                     uint32_t* __restrict__ drift_list,
                                                                     uint32_t* __restrict__ drift_count)
{
    StepParams s = s_in;
    fold_plain_model<FAST>(s);
    const uint64_t step_next = *step_ptr + 1;   // the step being produced (device-side counter: graph replays see it move)
    constexpr int CHUNK = TILD_INTERP_CHUNK, KCAP = TILD_INTERP_KCAP;
    extern __shared__ __align__(16) float fs[];
    __shared__ int goff_x[32], goff_y[32];
    __shared__ uint32_t cnt[32], novf, ndrift, drift_base;
    const int EX = tp.E[0];
    const int CS = EX * EY * EZ;                              // component stride of the image
    const int tile = blockIdx.x;
    const int tz = tile % tp.nt[2], ty = (tile / tp.nt[2]) % tp.nt[1], tx = tile / (tp.nt[2] * tp.nt[1]);
    const int o[3] = {tx * tp.T[0] - tp.lo, ty * tp.T[1] - tp.lo, tz * tp.T[2] - tp.lo - tp.sh};
    const int E[3] = {EX, tp.E[1], EZ};
    const size_t seg0 = (size_t)tile * m.S;
    if (seg_base[seg0] == seg_base[seg0 + m.S]) return;   // empty tile (uniform)
    uint16_t* idx = reinterpret_cast<uint16_t*>(fs + 3 * (size_t)CS);
    uint16_t* ovf = idx + KCAP * 32;
    if (threadIdx.x < EX) goff_x[threadIdx.x] = wrap_idx(o[0] + threadIdx.x, m.N[0]);
    else if (threadIdx.x >= 32 && threadIdx.x < 32 + EY) goff_y[threadIdx.x - 32] = wrap_idx(o[1] + threadIdx.x - 32, m.N[1]);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const bool vec16 = (m.N[2] % 4 == 0) && ((reinterpret_cast<uintptr_t>(ffield) & 15) == 0);

    for (int sp = 0; sp < m.S; ++sp) {
        const uint32_t p_lo = seg_base[seg0 + sp], p_hi = seg_base[seg0 + sp + 1];
        if (p_lo == p_hi) continue;                        // uniform
        __syncthreads();                                   // previous species' gathers are done; goff_* visible
        {
            // stage the field: one (x, y) column of the image per thread group, three components each
            const float* fsp = ffield + (size_t)sp * 3 * m.FM;
            if (vec16) {
                // 16-byte copies: the image starts on a 16-byte boundary of the mesh rows (tp.sh) and Nz % 4 == 0,
                // so every aligned float4 of a row stays inside the row and wraps as a whole
                constexpr int CPR = EZ / 4;                       // chunks per row
                constexpr int RPP = INTERP_THREADS / CPR;         // rows per pass
                const int chunk = threadIdx.x % CPR;
                const int gz = wrap_idx(o[2] + 4 * chunk, m.N[2]);
                if (threadIdx.x < RPP * CPR)
                    for (int q = threadIdx.x / CPR; q < EX * EY; q += RPP) {
                        const int lx = q / EY, ly = q - lx * EY;
                        if (ly >= E[1]) continue;
                        const float* src = fsp + ((size_t)goff_x[lx] * m.FN[0] + goff_y[ly]) * m.FN[1] + gz;
                        float* dst = fs + q * EZ + 4 * chunk;
#pragma unroll
                        for (int comp = 0; comp < 3; ++comp) cp_async_16(dst + comp * CS, src + (size_t)comp * m.FM);
                    }
            } else {
                constexpr int RPP = INTERP_THREADS / EZ;
                const int lz = threadIdx.x % EZ;
                const int gz = wrap_idx(o[2] + lz, m.N[2]);
                if (threadIdx.x < RPP * EZ)
                    for (int q = threadIdx.x / EZ; q < EX * EY; q += RPP) {
                        const int lx = q / EY, ly = q - lx * EY;
                        if (ly >= E[1]) continue;
                        const float* src = fsp + ((size_t)goff_x[lx] * m.FN[0] + goff_y[ly]) * m.FN[1] + gz;
                        float* dst = fs + q * EZ + lz;
#pragma unroll
                        for (int comp = 0; comp < 3; ++comp) cp_async_f32(dst + comp * CS, src + (size_t)comp * m.FM);
                    }
            }
            cp_async_commit();
        }
        for (uint32_t c0 = p_lo; c0 < p_hi; c0 += CHUNK) {
            const int nchunk = (int)min((uint32_t)CHUNK, p_hi - c0);
            // rounds reserved per class: a little above the mean; the rest is worked off in dense mixed rounds
            const uint32_t kcap = min((uint32_t)KCAP, (uint32_t)(nchunk + 31) / 32u + (uint32_t)(nchunk >> 9) + 1u);
            if (c0 != p_lo) __syncthreads();               // previous chunk's rounds are done
            if (threadIdx.x < 32) cnt[threadIdx.x] = 0u;
            if (threadIdx.x == 32) novf = 0u;
            if (threadIdx.x == 33) ndrift = 0u;
            __syncthreads();
            // phase A (overlaps the copies in flight): class = bank of the first stencil node in the image
            for (int i0 = threadIdx.x; i0 < nchunk; i0 += 3 * INTERP_THREADS) {   // three loads in flight per thread
                float4 pj[3];
#pragma unroll
                for (int j = 0; j < 3; ++j)
                    if (i0 + j * INTERP_THREADS < nchunk) pj[j] = X4[(size_t)c0 + i0 + j * INTERP_THREADS];
#pragma unroll
                for (int j = 0; j < 3; ++j) {
                const int i = i0 + j * INTERP_THREADS;
                if (i >= nchunk) break;
                const float4 p = pj[j];
                int b[3], d[3];
                float w[3][P];
                index_weights<P>(m, p, b, w);
                bool inside = true;
#pragma unroll
                for (int a = 0; a < 3; ++a) {
                    d[a] = wrap_near(b[a] - o[a], m.N[a]);
                    inside = inside && ((unsigned)d[a] + (unsigned)P <= (unsigned)E[a]);   // unsigned: a wild position (d < 0) is not inside
                }
                if (inside) {
                    const uint32_t cls = (uint32_t)((d[0] * EY + d[1]) * EZ + d[2]) & 31u;
                    const uint32_t k = atomicAdd(&cnt[cls], 1u);
                    if (k < kcap) idx[k * 32 + cls] = (uint16_t)i;
                    else ovf[atomicAdd(&novf, 1u)] = (uint16_t)i;
                } else {
                    // drifted out of the tile's halo since the last re-sort: queued (from the top of ovf) and done
                    // together after the rounds, so that one such particle does not stall the 31 other lanes here
                    ovf[CHUNK - 1 - atomicAdd(&ndrift, 1u)] = (uint16_t)i;
                }
                }
            }
            cp_async_wait_all();
            __syncthreads();
            // phase B: rounds of one particle per class, then the overflow (any class)
            const uint32_t mine = cnt[lane];
            uint32_t rounds = mine;
#pragma unroll
            for (int dlt = 16; dlt > 0; dlt >>= 1) rounds = max(rounds, __shfl_xor_sync(0xffffffffu, rounds, dlt));
            rounds = min(rounds, kcap);
            const uint32_t extra = (novf + 31u) >> 5;
            // software pipeline: the list entry and position of the NEXT round are fetched before this round's work
            auto fetch = [&](uint32_t k, int& i, float4& p) {
                i = -1;
                if (k < rounds) {
                    if (k < mine) i = idx[k * 32 + lane];
                } else if (k < rounds + extra) {
                    const uint32_t j = (k - rounds) * 32u + lane;
                    if (j < novf) i = ovf[j];
                }
                if (i >= 0) p = X4[(size_t)c0 + i];
            };
            int i_next;
            float4 p_next = make_float4(0.f, 0.f, 0.f, 0.f);
            fetch(wid, i_next, p_next);
            for (uint32_t k = wid; k < rounds + extra; k += INTERP_WARPS) {
                const int i = i_next;
                const float4 p = p_next;
                fetch(k + INTERP_WARPS, i_next, p_next);
                if (i < 0) continue;
                const size_t slot = (size_t)c0 + i;
                // issue the loads the finish needs now, so that their latency hides behind the stencil gather
                float4 w0 = make_float4(0.f, 0.f, 0.f, 0.f), q0 = p, q1 = p;
                int bj0 = -1, bj1 = -1;
                if (MODE == 2) w0 = W4[slot];
                if (MODE >= 1 && s.max_bonds == 2) {
                    const int2 bb = *reinterpret_cast<const int2*>(B + 2 * slot);
                    bj0 = bb.x;
                    bj1 = bb.y;
                } else if (MODE >= 1 && s.max_bonds == 1) {
                    bj0 = B[slot];
                }
                int b[3];
                float w[3][P];
                index_weights<P>(m, p, b, w);
                if (MODE >= 1 && bj0 >= 0) q0 = X4[bj0];
                if (MODE >= 1 && bj1 >= 0) q1 = X4[bj1];
                const float* f0 = fs + (wrap_near(b[0] - o[0], m.N[0]) * EY + wrap_near(b[1] - o[1], m.N[1])) * EZ +
                                  wrap_near(b[2] - o[2], m.N[2]);
                const float* f1 = f0 + CS;
                const float* f2 = f1 + CS;
                float3 F = make_float3(0.f, 0.f, 0.f);
#pragma unroll
                for (int jx = 0; jx < P; ++jx) {
#pragma unroll
                    for (int jy = 0; jy < P; ++jy) {
                        const int off = (jx * EY + jy) * EZ;
                        float tx_ = 0.f, ty_ = 0.f, tz_ = 0.f;
#pragma unroll
                        for (int jz = 0; jz < P; ++jz) {
                            tx_ = fmaf(w[2][jz], f0[off + jz], tx_);
                            ty_ = fmaf(w[2][jz], f1[off + jz], ty_);
                            tz_ = fmaf(w[2][jz], f2[off + jz], tz_);
                        }
                        const float wxy = w[0][jx] * w[1][jy];
                        F.x = fmaf(wxy, tx_, F.x);
                        F.y = fmaf(wxy, ty_, F.y);
                        F.z = fmaf(wxy, tz_, F.z);
                    }
                }
                if (MODE >= 1) {
                    if (s.max_bonds <= 2) {
                        if (bj0 >= 0) bond_term(m, s, p, q0, F);
                        if (bj1 >= 0) bond_term(m, s, p, q1, F);
                        if (s.lambda_wlc != 0.0f || s.k_theta != 0.0f) angle_force_slots(m, s, X4, B, slot, p, F);
                    } else {
                        const float3 fb = bond_force_slots(m, s, X4, B, slot, p);
                        F.x += fb.x;
                        F.y += fb.y;
                        F.z += fb.z;
                    }
                }
                finish_update<MODE>(m, s, step_next, slot, p, F, w0, X4o, W4o, F4);
            }
            // drifted particles of this chunk: handed to interp_drift_kernel through a global list (one global
            // atomic per chunk), so that their long global gathers are off this CTA's critical path
            if (ndrift > 0) {                              // uniform: ndrift is stable since the sync after phase A
                if (threadIdx.x == 0) drift_base = atomicAdd(drift_count, ndrift);
                __syncthreads();
                for (uint32_t j = threadIdx.x; j < ndrift; j += INTERP_THREADS)
                    drift_list[drift_base + j] = c0 + ovf[CHUNK - 1 - j];
            }
        }
    }
}

// particles that left their tile's image since the last re-sort: per-particle global gather, any order.
// Last kernel of the fused pass: the block that finishes last resets the drift counter for the next pass and, in the
// fused step (step_adv != nullptr), advances the device-side step counter -- no extra launches for either.
template <int P, int MODE, bool FAST>
__global__ void __launch_bounds__(256) interp_drift_kernel(MeshParams m, StepParams s_in, const uint64_t* step_ptr,
                                                           const uint32_t* __restrict__ drift_list,
                                                           uint32_t* __restrict__ drift_count, uint64_t* __restrict__ step_adv,
                                                           const float* __restrict__ ffield, const float4* __restrict__ X4,
                                                           const float4* __restrict__ W4, const int32_t* __restrict__ B,
                                                           float4* __restrict__ X4o, float4* __restrict__ W4o,
                                                           float4* __restrict__ F4, float4* __restrict__ zgrid, size_t zcount4)
{
    StepParams s = s_in;
    fold_plain_model<FAST>(s);
    // The density grid of the next step, cleared here instead of by a memset in front of the spread: this kernel waits on
    // gather latency and leaves HBM idle, so the stores are free (they drain while the gathers below are in flight).
    if (zgrid)
        for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < zcount4; i += (size_t)gridDim.x * blockDim.x)
            zgrid[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    const uint64_t step_next = *step_ptr + 1;   // the step being produced (device-side counter: graph replays see it move)
    const uint32_t nd = *drift_count;
    // G lanes share a particle (its P P stencil rows dealt round-robin): the kernel is bound by the latency of the gathers
    // (the field left L2 long ago), so what counts is how many of them are in flight
    constexpr int G = P >= 3 ? 8 : P == 2 ? 4 : 1;
    const bool vec = (m.N[2] % 4 == 0) && ((reinterpret_cast<uintptr_t>(ffield) & 15) == 0);   // uniform
    const uint32_t g = threadIdx.x % G, per_pass = gridDim.x * (blockDim.x / G);
    for (uint32_t j0 = 0; j0 < nd; j0 += per_pass) {                  // uniform trip count: the shuffles below are full-warp
        const uint32_t j = j0 + blockIdx.x * (blockDim.x / G) + threadIdx.x / G;
        const bool act = j < nd;
        const size_t slot = act ? drift_list[j] : 0;
        float4 p = make_float4(0.f, 0.f, 0.f, 0.f);
        float3 F = make_float3(0.f, 0.f, 0.f);
        if (act) {
            p = X4[slot];
            int b[3];
            float w[3][P];
            index_weights<P>(m, p, b, w);
            F = vec ? interp_global_rows<P, true, G>(m, ffield, b, w, __float_as_int(p.w), (int)g)
                    : interp_global_rows<P, false, G>(m, ffield, b, w, __float_as_int(p.w), (int)g);
        }
#pragma unroll
        for (int d = G / 2; d > 0; d >>= 1) {
            F.x += __shfl_xor_sync(0xffffffffu, F.x, d);
            F.y += __shfl_xor_sync(0xffffffffu, F.y, d);
            F.z += __shfl_xor_sync(0xffffffffu, F.z, d);
        }
        if (act && g == 0) finish_particle<MODE>(m, s, step_next, slot, p, F, X4, W4, B, X4o, W4o, F4);
    }
    __syncthreads();                            // every thread of this block has read the step and the drift count
    if (threadIdx.x == 0) {
        __threadfence();
        if (atomicAdd(drift_count + 1, 1u) == gridDim.x - 1) {   // all blocks are past their reads
            drift_count[0] = 0u;
            drift_count[1] = 0u;
            if (step_adv) *step_adv = step_next;
        }
    }
}

// caller-order bond force (stage call)
__global__ void __launch_bounds__(256) bond_force_kernel(MeshParams m, StepParams s, const float* __restrict__ x,
                                                         const int32_t* __restrict__ bond, float* __restrict__ f)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= m.n) return;
    const float px = x[3 * (size_t)i], py = x[3 * (size_t)i + 1], pz = x[3 * (size_t)i + 2];
    float3 acc = make_float3(0.f, 0.f, 0.f);
    for (int k = 0; k < s.max_bonds; ++k) {
        const int32_t j = bond[(size_t)i * s.max_bonds + k];
        if (j < 0) continue;
        const float dx = min_image(px - x[3 * (size_t)j + 0], m.L[0], m.inv_L[0]);
        const float dy = min_image(py - x[3 * (size_t)j + 1], m.L[1], m.inv_L[1]);
        const float dz = min_image(pz - x[3 * (size_t)j + 2], m.L[2], m.inv_L[2]);
        float scale = -2.0f * s.k_bond;
        if (s.r0_bond != 0.0f) {
            const float r = sqrtf(dx * dx + dy * dy + dz * dz);
            scale = r > 0.0f ? scale * (1.0f - s.r0_bond / r) : 0.0f;
        }
        acc.x += scale * dx;
        acc.y += scale * dy;
        acc.z += scale * dz;
    }
    if (s.lambda_wlc != 0.0f || s.k_theta != 0.0f) {   // angles, Eq. 16-17 (max_bonds == 2: slot 0 = previous, slot 1 = next bead)
        const int32_t jp = bond[2 * (size_t)i], jn = bond[2 * (size_t)i + 1];
        const float r[3] = {px, py, pz};
        float prev[3] = {0.f, 0.f, 0.f}, next[3] = {0.f, 0.f, 0.f}, pprev[3] = {0.f, 0.f, 0.f}, nnext[3] = {0.f, 0.f, 0.f};
        bool has_pprev = false, has_nnext = false;
        if (jp >= 0) {
            for (int a = 0; a < 3; ++a) prev[a] = x[3 * (size_t)jp + a];
            const int32_t pp = bond[2 * (size_t)jp];
            if (pp >= 0) {
                for (int a = 0; a < 3; ++a) pprev[a] = x[3 * (size_t)pp + a];
                has_pprev = true;
            }
        }
        if (jn >= 0) {
            for (int a = 0; a < 3; ++a) next[a] = x[3 * (size_t)jn + a];
            const int32_t nn = bond[2 * (size_t)jn + 1];
            if (nn >= 0) {
                for (int a = 0; a < 3; ++a) nnext[a] = x[3 * (size_t)nn + a];
                has_nnext = true;
            }
        }
        float fa[3] = {0.f, 0.f, 0.f};
        wlc_angle_force(s.lambda_wlc, s.k_theta, s.theta0, m.L, m.inv_L, r, jp >= 0, prev, has_pprev, pprev, jn >= 0, next, has_nnext, nnext, fa);
        acc.x += fa[0];
        acc.y += fa[1];
        acc.z += fa[2];
    }
    f[3 * (size_t)i + 0] = acc.x;
    f[3 * (size_t)i + 1] = acc.y;
    f[3 * (size_t)i + 2] = acc.z;
}

// w.xyz += alpha * f.xyz on occupied slots
__global__ void __launch_bounds__(256) axpy_slots_kernel(size_t nslots, float alpha, const float4* __restrict__ F4, float4* __restrict__ W4)
{
    const size_t s = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= nslots) return;
    float4 w = W4[s];
    const float4 f = F4[s];
    w.x += alpha * f.x;
    w.y += alpha * f.y;
    w.z += alpha * f.z;
    W4[s] = w;
}

// v[id] = w + alpha f
__global__ void __launch_bounds__(256) velocity_out_kernel(size_t nslots, float alpha, const float4* __restrict__ F4,
                                                           const float4* __restrict__ W4, float* __restrict__ v)
{
    const size_t s = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= nslots) return;
    const float4 w = W4[s];
    const uint32_t id = __float_as_uint(w.w);
    const float4 f = alpha != 0.0f ? F4[s] : make_float4(0.f, 0.f, 0.f, 0.f);
    v[3 * (size_t)id + 0] = w.x + alpha * f.x;
    v[3 * (size_t)id + 1] = w.y + alpha * f.y;
    v[3 * (size_t)id + 2] = w.z + alpha * f.z;
}

__global__ void philox_test_kernel(int m, const uint32_t* __restrict__ ctr, const uint32_t* __restrict__ key,
                                   uint32_t* __restrict__ out, float* __restrict__ gauss)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= m) return;
    const uint4 c = make_uint4(ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3]);
    const uint4 r = philox4x32_10(c, key[2 * i], key[2 * i + 1]);
    out[4 * i] = r.x;
    out[4 * i + 1] = r.y;
    out[4 * i + 2] = r.z;
    out[4 * i + 3] = r.w;
    if (gauss) {
        const float3 z = gauss3(c.x, (uint64_t)c.y | ((uint64_t)c.z << 32), key[2 * i], key[2 * i + 1]);
        gauss[3 * i] = z.x;
        gauss[3 * i + 1] = z.y;
        gauss[3 * i + 2] = z.z;
    }
}

bool can_vectorize(const tild_ctx* c, const float* ffield)
{
    return (c->mesh.N[2] % 4 == 0) && (reinterpret_cast<uintptr_t>(ffield) % 16 == 0);
}

// ---- dispatch ------------------------------------------------------------------------------------------------------

template <int P, int EY, int EZ, int MODE, bool FAST>
void tile_launch(const InterpArgs& a, cudaStream_t st, size_t smem, bool configure_only, cudaError_t* err)
{
    auto kernel = interp_tile_kernel<P, EY, EZ, MODE, FAST>;
    if (configure_only) {
        const cudaError_t e = tild_raise_smem_limit(reinterpret_cast<const void*>(kernel), smem);
        if (e != cudaSuccess) *err = e;
        return;
    }
    kernel<<<a.tp.ntiles, INTERP_THREADS, smem, st>>>(a.m, a.tp, a.s, a.step_ptr, a.seg_base, a.ffield, a.X4, a.W4, a.B, a.X4o,
                                                      a.W4o, a.F4, a.drift_list, a.drift_count);
    interp_drift_kernel<P, MODE, FAST><<<1184, 256, 0, st>>>(a.m, a.s, a.step_ptr, a.drift_list, a.drift_count, MODE == 2 ? a.step_adv : nullptr,
                                                            a.ffield, a.X4, a.W4, a.B, a.X4o, a.W4o, a.F4, MODE == 2 ? a.zgrid : nullptr, a.zcount4);
}
template <int P, int EY, int EZ>
void tile_launch_m(const InterpArgs& a, int mode, cudaStream_t st, size_t smem, bool cfg, cudaError_t* err)
{
    const bool fast = plain_model(a.s);
    if (cfg || mode == 0) tile_launch<P, EY, EZ, 0, false>(a, st, smem, cfg, err);
    if (cfg || mode == 1) tile_launch<P, EY, EZ, 1, false>(a, st, smem, cfg, err);
    if (cfg || (mode == 2 && !fast)) tile_launch<P, EY, EZ, 2, false>(a, st, smem, cfg, err);
    if (cfg || (mode == 2 && fast)) tile_launch<P, EY, EZ, 2, true>(a, st, smem, cfg, err);
}
template <int P>
bool tile_launch_p(const InterpArgs& a, int ey, int ez, int mode, cudaStream_t st, size_t smem, bool cfg, cudaError_t* err)
{
    constexpr int H = Halo<P>::H, EZA = Halo<P>::EZA, EZB = Halo<P>::EZB;
    if (ey == 8 + H && ez == EZA) tile_launch_m<P, 8 + H, EZA>(a, mode, st, smem, cfg, err);
    else if (ey == 8 + H && ez == EZB) tile_launch_m<P, 8 + H, EZB>(a, mode, st, smem, cfg, err);
    else if (ey == 16 + H && ez == EZA) tile_launch_m<P, 16 + H, EZA>(a, mode, st, smem, cfg, err);
    else if (ey == 16 + H && ez == EZB) tile_launch_m<P, 16 + H, EZB>(a, mode, st, smem, cfg, err);
    else return false;
    return true;
}
bool tile_launch_any(const InterpArgs& a, int mode, cudaStream_t st, size_t smem, bool cfg, cudaError_t* err)
{
    switch (a.m.P) {
    case 1: return tile_launch_p<1>(a, a.tp.EY, a.tp.EZ, mode, st, smem, cfg, err);
    case 2: return tile_launch_p<2>(a, a.tp.EY, a.tp.EZ, mode, st, smem, cfg, err);
    case 3: return tile_launch_p<3>(a, a.tp.EY, a.tp.EZ, mode, st, smem, cfg, err);
    case 4: return tile_launch_p<4>(a, a.tp.EY, a.tp.EZ, mode, st, smem, cfg, err);
    default: return tile_launch_p<5>(a, a.tp.EY, a.tp.EZ, mode, st, smem, cfg, err);
    }
}

// the drifted particles of the rotation-class kernel (P = 4)
void launch_drift_only(const InterpArgs& a, int mode, cudaStream_t st)
{
#define TILD_DR(M_, F_) interp_drift_kernel<4, M_, F_><<<1184, 256, 0, st>>>(a.m, a.s, a.step_ptr, a.drift_list, a.drift_count, M_ == 2 ? a.step_adv : nullptr, a.ffield, a.X4, a.W4, a.B, a.X4o, a.W4o, a.F4, M_ == 2 ? a.zgrid : nullptr, a.zcount4)
    if (mode == 0) TILD_DR(0, false); else if (mode == 1) TILD_DR(1, false); else if (plain_model(a.s)) TILD_DR(2, true); else TILD_DR(2, false);
#undef TILD_DR
}

template <int P>
void slots_launch_p(const InterpArgs& a, bool vec, int mode, size_t s0, size_t s1, cudaStream_t st)
{
    const unsigned nb = (unsigned)((s1 - s0 + 255) / 256);
#define TILD_SL(V, M_, F_) interp_slots_kernel<P, V, M_, F_><<<nb, 256, 0, st>>>(a.m, a.s, a.step_ptr, s0, s1, a.ffield, a.X4, a.W4, a.B, a.X4o, a.W4o, a.F4)
    const bool fast = plain_model(a.s);
    if (vec) { if (mode == 0) TILD_SL(true, 0, false); else if (mode == 1) TILD_SL(true, 1, false); else if (fast) TILD_SL(true, 2, true); else TILD_SL(true, 2, false); }
    else     { if (mode == 0) TILD_SL(false, 0, false); else if (mode == 1) TILD_SL(false, 1, false); else if (fast) TILD_SL(false, 2, true); else TILD_SL(false, 2, false); }
#undef TILD_SL
}

}  // namespace

int tild_interp_configure(tild_ctx* c)
{
    if (!c->tile.enabled) return TILD_OK;
    InterpArgs a{};
    a.m = c->mesh;
    a.tp = c->tile;
    cudaError_t e = cudaSuccess;
    if (interp_rot_applies(c)) {
        interp_rot_make_tmap(c);
        e = interp_rot_run(a, 0, c->stream, true);
        if (e != cudaSuccess)
            return tild_fail(c, TILD_ECUDA, "cudaFuncSetAttribute(interp_rot_kernel): %s", cudaGetErrorString(e));
    }
    if (!tile_launch_any(a, 0, c->stream, c->tile.smem_interp, true, &e))
        return tild_fail(c, TILD_EINVAL, "no interp tile kernel for P=%d EY=%d EZ=%d", c->mesh.P, c->tile.EY, c->tile.EZ);
    if (e != cudaSuccess)
        return tild_fail(c, TILD_ECUDA, "cudaFuncSetAttribute(interp_tile_kernel, %zu B): %s", c->tile.smem_interp, cudaGetErrorString(e));
    return TILD_OK;
}

int launch_interp(tild_ctx* c, int mode, const SegLayout& lay, const float* ffield, const float4* X4, const float4* W4,
                  const int32_t* B, float4* X4o, float4* W4o, float* /*unused*/)
{
    const size_t n = (size_t)c->mesh.n;
    if (n == 0) return TILD_OK;
    InterpArgs a{c->mesh, c->tile, c->stp, c->d_step, lay.seg_base, ffield, X4, W4, B, X4o, W4o, c->F4, c->rank, c->drift_count, c->d_step,
                 c->fmap, (c->tma_ok && ffield == c->ffield) ? 1 : 0,    // the tensor map describes the library's own field
                 nullptr, 0};
    c->step_advanced = false;
    if (c->tile.enabled && c->mesh.P >= 2 && !(c->prm.flags & TILD_FLAG_NAIVE_INTERP)) {   // P = 1: one node per particle
        cudaError_t e = cudaSuccess;
        // drift_count[0..1] are zero here: cleared at tild_init and again by the last block of every drift kernel
        c->step_advanced = mode == INTERP_FUSED_STEP;
        const size_t gridf = c->M * (size_t)c->mesh.S;
        if (mode == INTERP_FUSED_STEP && gridf % 4 == 0 && (reinterpret_cast<uintptr_t>(c->grid) & 15) == 0) {
            a.zgrid = reinterpret_cast<float4*>(c->grid);   // dead since the forward transform of this step
            a.zcount4 = gridf / 4;
        }
        if (interp_rot_applies(c) && !(c->prm.flags & TILD_FLAG_GEN1_TILES)) {
            e = interp_rot_run(a, mode, c->stream, false);
            TILD_LAUNCH_CHECK(c, "interp_rot_kernel");
            InterpArgs ad = a;
            ad.zgrid = nullptr;                            // the tile kernel has cleared the grid
            launch_drift_only(ad, mode, c->stream);
        } else {
            tile_launch_any(a, mode, c->stream, c->tile.smem_interp, false, &e);
            TILD_LAUNCH_CHECK(c, "interp_tile_kernel");
        }
        TILD_LAUNCH_CHECK(c, "interp_drift_kernel");
        if (a.zgrid) c->grid_clean = true;
        return TILD_OK;
    }
    const bool vec = can_vectorize(c, ffield);
    switch (c->mesh.P) {
    case 1: slots_launch_p<1>(a, vec, mode, 0, n, c->stream); break;
    case 2: slots_launch_p<2>(a, vec, mode, 0, n, c->stream); break;
    case 3: slots_launch_p<3>(a, vec, mode, 0, n, c->stream); break;
    case 4: slots_launch_p<4>(a, vec, mode, 0, n, c->stream); break;
    default: slots_launch_p<5>(a, vec, mode, 0, n, c->stream); break;
    }
    TILD_LAUNCH_CHECK(c, "interp_slots_kernel");
    return TILD_OK;
}

__global__ void advance_step_kernel(uint64_t* step) { *step += 1; }

int launch_advance_step(tild_ctx* c)
{
    advance_step_kernel<<<1, 1, 0, c->stream>>>(c->d_step);
    TILD_LAUNCH_CHECK(c, "advance_step_kernel");
    return TILD_OK;
}

int launch_bond_force_caller(tild_ctx* c, const float* x, const int32_t* bond, float* f)
{
    const int n = c->mesh.n;
    if (n == 0) return TILD_OK;
    bond_force_kernel<<<(n + 255) / 256, 256, 0, c->stream>>>(c->mesh, c->stp, x, bond, f);
    TILD_LAUNCH_CHECK(c, "bond_force_kernel");
    return TILD_OK;
}

int launch_make_w(tild_ctx* c, const float4* F4, float4* W4, float sign)
{
    const size_t nslots = (size_t)c->mesh.n;
    if (nslots == 0) return TILD_OK;
    axpy_slots_kernel<<<(unsigned)((nslots + 255) / 256), 256, 0, c->stream>>>(nslots, sign * c->stp.half_dt_over_m, F4, W4);
    TILD_LAUNCH_CHECK(c, "axpy_slots_kernel");
    return TILD_OK;
}

int launch_velocity_out(tild_ctx* c, const float4* F4, const float4* W4, float* v)
{
    const size_t nslots = (size_t)c->mesh.n;
    if (nslots == 0) return TILD_OK;
    velocity_out_kernel<<<(unsigned)((nslots + 255) / 256), 256, 0, c->stream>>>(nslots, c->stp.kick_in, F4, W4, v);
    TILD_LAUNCH_CHECK(c, "velocity_out_kernel");
    return TILD_OK;
}

int launch_philox_test(tild_ctx* c, const uint32_t* ctr, const uint32_t* key, uint32_t* out, float* gauss, int m)
{
    if (m <= 0) return TILD_OK;
    philox_test_kernel<<<(m + 127) / 128, 128, 0, c->stream>>>(m, ctr, key, out, gauss);
    TILD_LAUNCH_CHECK(c, "philox_test_kernel");
    return TILD_OK;
}
