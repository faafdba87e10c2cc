// Per-particle device helpers shared by the interpolation kernels (tild_interp.cu, tild_interp_rot.cu):
// global gather of the stencil, bond / angle forces (Eq. 2, Eq. 16-17) and the
// integrator update (GJF L352 / Euler-Maruyama L348; A11, A11b).  Internal; not part of the C-ABI.
#pragma once
#include "tild_internal.cuh"

namespace {

// ---- per-particle global gather (overflow tail, drifted particles, grids too small for tiles) -------------------
// VEC = true (Nz % 4 == 0, 16-byte aligned field): the P nodes of one z-row are contiguous in memory but start at
// an arbitrary z, so each row is read as the one or two ALIGNED float4 that cover it (LDG.128) and dotted with an
// 8-wide weight vector holding w_z shifted to the row's offset and zeros elsewhere.
template <int P, bool VEC>
__device__ __forceinline__ float3 interp_global(const MeshParams& m, const float* __restrict__ ffield, const int b[3],
                                                const float w[3][P], int type)
{
    const float* fx = ffield + (size_t)type * 3 * m.FM;
    const float* fy = fx + m.FM;
    const float* fz = fy + m.FM;
    float3 acc = make_float3(0.f, 0.f, 0.f);
    if (VEC) {
        const int bzw = wrap_idx(b[2], m.N[2]);
        const int a0 = bzw & ~3, off = bzw & 3;
        const int a1 = (a0 + 4 >= m.N[2]) ? 0 : a0 + 4;
        const bool two = off + P > 4;
        float w8[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            float v = 0.f;
#pragma unroll
            for (int j = 0; j < P; ++j)
                if (k - j >= 0 && k - j <= 3) v = (k - j == off) ? w[2][j] : v;
            w8[k] = v;
        }
#pragma unroll
        for (int jx = 0; jx < P; ++jx) {
            const size_t ox = (size_t)wrap_idx(b[0] + jx, m.N[0]) * m.FN[0];
#pragma unroll
            for (int jy = 0; jy < P; ++jy) {
                const size_t row = (ox + wrap_idx(b[1] + jy, m.N[1])) * m.FN[1];
                const float wxy = w[0][jx] * w[1][jy];
                const float* comp[3] = {fx, fy, fz};
                float d[3];
#pragma unroll
                for (int q = 0; q < 3; ++q) {
                    const float4 v0 = __ldg(reinterpret_cast<const float4*>(comp[q] + row + a0));
                    float s = w8[0] * v0.x + w8[1] * v0.y + w8[2] * v0.z + w8[3] * v0.w;
                    if (two) {
                        const float4 v1 = __ldg(reinterpret_cast<const float4*>(comp[q] + row + a1));
                        s += w8[4] * v1.x + w8[5] * v1.y + w8[6] * v1.z + w8[7] * v1.w;
                    }
                    d[q] = s;
                }
                acc.x += wxy * d[0];
                acc.y += wxy * d[1];
                acc.z += wxy * d[2];
            }
        }
        return acc;
    }
    int iz[P];
#pragma unroll
    for (int j = 0; j < P; ++j) iz[j] = wrap_idx(b[2] + j, m.N[2]);
#pragma unroll
    for (int jx = 0; jx < P; ++jx) {
        const size_t ox = (size_t)wrap_idx(b[0] + jx, m.N[0]) * m.FN[0];
#pragma unroll
        for (int jy = 0; jy < P; ++jy) {
            const size_t row = (ox + wrap_idx(b[1] + jy, m.N[1])) * m.FN[1];
            const float wxy = w[0][jx] * w[1][jy];
#pragma unroll
            for (int jz = 0; jz < P; ++jz) {
                const float ww = wxy * w[2][jz];
                const size_t g = row + iz[jz];
                acc.x += ww * __ldg(fx + g);
                acc.y += ww * __ldg(fy + g);
                acc.z += ww * __ldg(fz + g);
            }
        }
    }
    return acc;
}

// The (x, y) rows r0, r0 + G, ... (< P P) of one particle's stencil: one lane of a group of G lanes that share a particle
// (interp_drift_kernel); the group's partial sums are added by the caller.
template <int P, bool VEC, int G>
__device__ __forceinline__ float3 interp_global_rows(const MeshParams& m, const float* __restrict__ ffield, const int b[3],
                                                     const float w[3][P], int type, int r0)
{
    const float* comp[3];
    comp[0] = ffield + (size_t)type * 3 * m.FM;
    comp[1] = comp[0] + m.FM;
    comp[2] = comp[1] + m.FM;
    float acc[3] = {0.f, 0.f, 0.f};
    const int bzw = wrap_idx(b[2], m.N[2]);
    const int a0 = bzw & ~3, off = bzw & 3;
    const int a1 = (a0 + 4 >= m.N[2]) ? 0 : a0 + 4;
    const bool two = off + P > 4;
    float w8[8];
    int iz[P];
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        float v = 0.f;
#pragma unroll
        for (int j = 0; j < P; ++j)
            if (k - j >= 0 && k - j <= 3) v = (k - j == off) ? w[2][j] : v;
        w8[k] = v;
    }
#pragma unroll
    for (int j = 0; j < P; ++j) iz[j] = wrap_idx(b[2] + j, m.N[2]);
#pragma unroll
    for (int i = 0; i < (P * P + G - 1) / G; ++i) {
        const int r = r0 + i * G;
        if (r >= P * P) break;
        const int jx = r / P, jy = r - jx * P;
        float wx = w[0][0], wy = w[1][0];
#pragma unroll
        for (int j = 1; j < P; ++j) {
            wx = jx == j ? w[0][j] : wx;
            wy = jy == j ? w[1][j] : wy;
        }
        const size_t row = ((size_t)wrap_idx(b[0] + jx, m.N[0]) * m.FN[0] + wrap_idx(b[1] + jy, m.N[1])) * m.FN[1];
        const float wxy = wx * wy;
#pragma unroll
        for (int q = 0; q < 3; ++q) {
            float sum = 0.f;
            if (VEC) {
                const float4 v0 = __ldg(reinterpret_cast<const float4*>(comp[q] + row + a0));
                sum = w8[0] * v0.x + w8[1] * v0.y + w8[2] * v0.z + w8[3] * v0.w;
                if (two) {
                    const float4 v1 = __ldg(reinterpret_cast<const float4*>(comp[q] + row + a1));
                    sum += w8[4] * v1.x + w8[5] * v1.y + w8[6] * v1.z + w8[7] * v1.w;
                }
            } else {
#pragma unroll
                for (int jz = 0; jz < P; ++jz) sum += w[2][jz] * __ldg(comp[q] + row + iz[jz]);
            }
            acc[q] += wxy * sum;
        }
    }
    return make_float3(acc[0], acc[1], acc[2]);
}

// The plain model of the BASELINE configs: two bond slots, no rest length, no angle potentials, three dimensions, an inertial
// integrator (GJF or VV + Langevin: one code path, other coefficients).  Kernels instantiated with FAST fold these facts in
// at compile time (fold_plain_model), which removes the call sites of the generic routines and their never-taken branches.
inline bool plain_model(const StepParams& s)
{
    return s.max_bonds == 2 && s.r0_bond == 0.0f && s.lambda_wlc == 0.0f && s.k_theta == 0.0f && !s.dim2 && s.integrator != TILD_INTEGRATOR_EM;
}
template <bool FAST>
__device__ __forceinline__ void fold_plain_model(StepParams& s)
{
    if (FAST) {
        s.max_bonds = 2;
        s.r0_bond = 0.0f;
        s.lambda_wlc = 0.0f;
        s.k_theta = 0.0f;
        s.dim2 = 0;
        s.integrator = TILD_INTEGRATOR_GJF;
    }
}

// f += force on the particle at p from the bond to the particle at q (Eq. 2; minimum image)
__device__ __forceinline__ void bond_term(const MeshParams& m, const StepParams& s, const float4& p, const float4& q, float3& f)
{
    const float dx = min_image(p.x - q.x, m.L[0], m.inv_L[0]);
    const float dy = min_image(p.y - q.y, m.L[1], m.inv_L[1]);
    const float dz = min_image(p.z - q.z, m.L[2], m.inv_L[2]);
    float scale = -2.0f * s.k_bond;
    if (s.r0_bond != 0.0f) {
        const float r = sqrtf(dx * dx + dy * dy + dz * dz);
        scale = r > 0.0f ? scale * (1.0f - s.r0_bond / r) : 0.0f;
    }
    f.x += scale * dx;
    f.y += scale * dy;
    f.z += scale * dz;
}

// f += cosine angle force (Eq. 16; max_bonds == 2: slot 0 = previous bead, slot 1 = next bead, A23)
__device__ __noinline__ void angle_force_slots(const MeshParams& m, const StepParams& s, const float4* __restrict__ X4,
                                                  const int32_t* __restrict__ B, size_t slot, const float4& p, float3& f)
{
    const int2 bb = *reinterpret_cast<const int2*>(B + 2 * slot);
    const float r[3] = {p.x, p.y, p.z};
    float prev[3] = {0.f, 0.f, 0.f}, next[3] = {0.f, 0.f, 0.f}, pprev[3] = {0.f, 0.f, 0.f}, nnext[3] = {0.f, 0.f, 0.f};
    bool has_pprev = false, has_nnext = false;
    if (bb.x >= 0) {
        const float4 q = X4[bb.x];
        prev[0] = q.x; prev[1] = q.y; prev[2] = q.z;
        const int32_t pp = B[2 * (size_t)bb.x];
        if (pp >= 0) {
            const float4 qq = X4[pp];
            pprev[0] = qq.x; pprev[1] = qq.y; pprev[2] = qq.z;
            has_pprev = true;
        }
    }
    if (bb.y >= 0) {
        const float4 q = X4[bb.y];
        next[0] = q.x; next[1] = q.y; next[2] = q.z;
        const int32_t nn = B[2 * (size_t)bb.y + 1];
        if (nn >= 0) {
            const float4 qq = X4[nn];
            nnext[0] = qq.x; nnext[1] = qq.y; nnext[2] = qq.z;
            has_nnext = true;
        }
    }
    float fa[3] = {0.f, 0.f, 0.f};
    wlc_angle_force(s.lambda_wlc, s.k_theta, s.theta0, m.L, m.inv_L, r, bb.x >= 0, prev, has_pprev, pprev, bb.y >= 0, next, has_nnext, nnext, fa);
    f.x += fa[0];
    f.y += fa[1];
    f.z += fa[2];
}

// Bond force on the particle at p from its partners' positions (slots into X4).
__device__ __noinline__ float3 bond_force_slots(const MeshParams& m, const StepParams& s, const float4* __restrict__ X4,
                                                   const int32_t* __restrict__ B, size_t slot, const float4& p)
{
    float3 f = make_float3(0.f, 0.f, 0.f);
    for (int k = 0; k < s.max_bonds; ++k) {
        const int32_t j = B[slot * s.max_bonds + k];
        if (j >= 0) bond_term(m, s, p, X4[j], f);
    }
    if (s.lambda_wlc != 0.0f || s.k_theta != 0.0f) angle_force_slots(m, s, X4, B, slot, p, f);
    return f;
}

// What happens to one particle once its interpolated force is known.
//   MODE 0: F4[slot] = interpolated force            (stage call tild_interp)
//   MODE 1: F4[slot] = interpolated + bond force     (tild_set_state / tild_get_state)
//   MODE 2: one GJF step: state (r^n, w^n), w^n = v^n - (dt/2m) F^n.
//     F^n = interp(r^n) + bonds(r^n);  v^n = w^n + (dt/2m) F^n;  beta = beta^{n+1} (Philox: id, step n+1)
//     r^{n+1} = wrap(r^n + b dt v^n + (b dt^2/2m) F^n + (b dt/2m) beta)
//     w^{n+1} = a v^n + (dt/2m) a F^n + (b/m) beta
//   Positions are double-buffered because bonds read the partners' r^n while r^{n+1} is written.
// F already holds the total force; w0 = W4[slot] (MODE 2 only)
template <int MODE>
__device__ __forceinline__ void finish_update(const MeshParams& m, const StepParams& s, uint64_t step_next, size_t slot,
                                              const float4& p, const float3& Fin, const float4& w0, float4* __restrict__ X4o,
                                              float4* __restrict__ W4o, float4* __restrict__ F4)
{
    float3 F = Fin;
    if (s.dim2) F.z = 0.0f;                      // A27: two-dimensional system, nothing acts or moves along z
    if (MODE <= 1) {
        F4[slot] = make_float4(F.x, F.y, F.z, 0.f);
        return;
    }
    float3 beta = make_float3(0.f, 0.f, 0.f);
    if (s.noise_amp != 0.0f) {
        const float3 z = gauss3(__float_as_uint(w0.w), step_next, s.key0, s.key1);
        beta = make_float3(s.noise_amp * z.x, s.noise_amp * z.y, s.dim2 ? 0.f : s.noise_amp * z.z);
    }
    if (s.integrator == TILD_INTEGRATOR_EM) {   // r' = r + (dt/gamma) F + beta/gamma; velocities are not used (A11b)
        X4o[slot] = make_float4(wrap_pos(p.x + (s.em_drift * F.x + s.em_noise * beta.x), m.L[0], m.inv_L[0]),
                                wrap_pos(p.y + (s.em_drift * F.y + s.em_noise * beta.y), m.L[1], m.inv_L[1]),
                                s.dim2 ? p.z : wrap_pos(p.z + (s.em_drift * F.z + s.em_noise * beta.z), m.L[2], m.inv_L[2]), p.w);
        W4o[slot] = w0;
        return;
    }
    const float pp[3] = {p.x, p.y, p.z};
    const float wv[3] = {w0.x, w0.y, w0.z};
    const float Fv[3] = {F.x, F.y, F.z};
    const float bv[3] = {beta.x, beta.y, beta.z};
    float xo[3], wo[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const float v = wv[a] + s.kick_in * Fv[a];
        const float r = pp[a] + (s.b_dt * v + s.b_dt2_over_2m * Fv[a] + s.b_dt_over_2m * bv[a]);
        xo[a] = wrap_pos(r, m.L[a], m.inv_L[a]);
        wo[a] = s.a_g * (v + s.w_fr * Fv[a]) + s.b_over_m * bv[a];
    }
    if (s.dim2) {
        xo[2] = p.z;
        wo[2] = 0.0f;
    }
    X4o[slot] = make_float4(xo[0], xo[1], xo[2], p.w);
    W4o[slot] = make_float4(wo[0], wo[1], wo[2], w0.w);
}

template <int MODE>
__device__ __forceinline__ void finish_particle(const MeshParams& m, const StepParams& s, uint64_t step_next, size_t slot,
                                                const float4& p, float3 F, const float4* __restrict__ X4,
                                                const float4* __restrict__ W4, const int32_t* __restrict__ B,
                                                float4* __restrict__ X4o, float4* __restrict__ W4o, float4* __restrict__ F4)
{
    float4 w0 = make_float4(0.f, 0.f, 0.f, 0.f);
    if (MODE == 2) w0 = W4[slot];
    if (MODE >= 1) {
        if (s.max_bonds == 2 && s.lambda_wlc == 0.0f && s.k_theta == 0.0f) {   // linear chains without angles: inline, no call
            const int2 bb = *reinterpret_cast<const int2*>(B + 2 * slot);
            const float4 q0 = X4[bb.x >= 0 ? (size_t)bb.x : slot], q1 = X4[bb.y >= 0 ? (size_t)bb.y : slot];   // self: zero force
            bond_term(m, s, p, q0, F);
            bond_term(m, s, p, q1, F);
        } else if (s.max_bonds > 0) {
            const float3 fb = bond_force_slots(m, s, X4, B, slot, p);          // generic tables, angle potentials (not inlined)
            F.x += fb.x;
            F.y += fb.y;
            F.z += fb.z;
        }
    }
    finish_update<MODE>(m, s, step_next, slot, p, F, w0, X4o, W4o, F4);
}

template <int P>
__device__ __forceinline__ void index_weights(const MeshParams& m, const float4& p, int b[3], float w[3][P])
{
    const float pos[3] = {p.x, p.y, p.z};
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        int cell;
        float t;
        index_1d<P>(pos[a], m.inv_h[a], cell, b[a], t);
        weights_1d<P>(t, w[a]);
    }
}

}  // namespace
