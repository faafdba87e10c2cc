// a6: mesh -> particle interpolation with the same weights (Fig. 1),
// harmonic bonds computed per particle without Newton's third law (Eq. 2) and the GJF Langevin
// update (L352; equations per DESIGN.md A11) fused into one pass over the particles.
#include "tild_internal.cuh"

namespace {

// f_a = sum_{stencil} w_x w_y w_z ffield[type][a][g]
//
// VEC = true (Nz % 4 == 0, 16-byte aligned field): the P nodes of one z-row are contiguous in memory but start at
// an arbitrary z, so each row is read as the one or two ALIGNED float4 that cover it (LDG.128) and dotted with an
// 8-wide weight vector holding w_z shifted to the row's offset and zeros elsewhere.  That halves the load
// instructions of the scalar form; with the particles in tile-major cell order (z fastest) the lanes of a warp
// read neighbouring z of the same rows, so each load touches few cache lines.
template <int P, bool VEC>
__device__ __forceinline__ float3 interp_one(const MeshParams& m, const float* __restrict__ ffield, float px, float py,
                                             float pz, int type)
{
    int cell, b[3];
    float t, w[3][P];
    index_1d<P>(px, m.inv_h[0], cell, b[0], t);
    weights_1d<P>(t, w[0]);
    index_1d<P>(py, m.inv_h[1], cell, b[1], t);
    weights_1d<P>(t, w[1]);
    index_1d<P>(pz, m.inv_h[2], cell, b[2], t);
    weights_1d<P>(t, w[2]);
    const float* fx = ffield + (size_t)type * 3 * m.M;
    const float* fy = fx + m.M;
    const float* fz = fy + m.M;
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
            const size_t ox = (size_t)wrap_idx(b[0] + jx, m.N[0]) * m.N[1];
#pragma unroll
            for (int jy = 0; jy < P; ++jy) {
                const size_t row = (ox + wrap_idx(b[1] + jy, m.N[1])) * m.N[2];
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
        const size_t ox = (size_t)wrap_idx(b[0] + jx, m.N[0]) * m.N[1];
#pragma unroll
        for (int jy = 0; jy < P; ++jy) {
            const size_t row = (ox + wrap_idx(b[1] + jy, m.N[1])) * m.N[2];
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

__device__ __forceinline__ float3 bond_force_one(const MeshParams& m, const StepParams& s, const float* __restrict__ x,
                                                 const int32_t* __restrict__ bond, size_t i, float px, float py, float pz)
{
    float3 f = make_float3(0.f, 0.f, 0.f);
    for (int k = 0; k < s.max_bonds; ++k) {
        const int32_t j = bond[i * s.max_bonds + k];
        if (j < 0) continue;
        const float dx = min_image(px - x[3 * (size_t)j + 0], m.L[0], m.inv_L[0]);
        const float dy = min_image(py - x[3 * (size_t)j + 1], m.L[1], m.inv_L[1]);
        const float dz = min_image(pz - x[3 * (size_t)j + 2], m.L[2], m.inv_L[2]);
        float scale = -2.0f * s.k_bond;
        if (s.r0_bond != 0.0f) {
            const float r = sqrtf(dx * dx + dy * dy + dz * dz);
            scale = r > 0.0f ? scale * (1.0f - s.r0_bond / r) : 0.0f;
        }
        f.x += scale * dx;
        f.y += scale * dy;
        f.z += scale * dz;
    }
    return f;
}

template <int P, bool VEC>
__global__ void __launch_bounds__(256) interp_force_kernel(MeshParams m, const float* __restrict__ ffield,
                                                           const float* __restrict__ x, const int32_t* __restrict__ type,
                                                           float* __restrict__ f)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= m.n) return;
    const float3 a = interp_one<P, VEC>(m, ffield, x[3 * (size_t)i], x[3 * (size_t)i + 1], x[3 * (size_t)i + 2], type[i]);
    f[3 * (size_t)i + 0] = a.x;
    f[3 * (size_t)i + 1] = a.y;
    f[3 * (size_t)i + 2] = a.z;
}

__global__ void __launch_bounds__(256) bond_force_kernel(MeshParams m, StepParams s, const float* __restrict__ x,
                                                         const int32_t* __restrict__ bond, float* __restrict__ f,
                                                         int accumulate)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= m.n) return;
    const float3 b = bond_force_one(m, s, x, bond, (size_t)i, x[3 * (size_t)i], x[3 * (size_t)i + 1], x[3 * (size_t)i + 2]);
    if (accumulate) {
        f[3 * (size_t)i + 0] += b.x;
        f[3 * (size_t)i + 1] += b.y;
        f[3 * (size_t)i + 2] += b.z;
    } else {
        f[3 * (size_t)i + 0] = b.x;
        f[3 * (size_t)i + 1] = b.y;
        f[3 * (size_t)i + 2] = b.z;
    }
}

// One pass per step n: state (r^n, w^n), w^n = v^n - (dt/2m) F^n.
//   F^n = interp(r^n) + bonds(r^n);  v^n = w^n + (dt/2m) F^n;  beta = beta^{n+1} (Philox: id, step n+1)
//   r^{n+1} = wrap(r^n + b dt v^n + (b dt^2/2m) F^n + (b dt/2m) beta)
//   w^{n+1} = a v^n + (dt/2m) a F^n + (b/m) beta
// Positions are double-buffered because bonds read the partners' r^n while r^{n+1} is written.
template <int P, bool VEC>
__global__ void __launch_bounds__(256) fused_step_kernel(MeshParams m, StepParams s, uint64_t step_next,
                                                         const float* __restrict__ ffield, const float* __restrict__ x0,
                                                         const float* __restrict__ w0, const int32_t* __restrict__ type,
                                                         const uint32_t* __restrict__ id, const int32_t* __restrict__ bond,
                                                         float* __restrict__ x1, float* __restrict__ w1)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= m.n) return;
    const float px = x0[3 * (size_t)i], py = x0[3 * (size_t)i + 1], pz = x0[3 * (size_t)i + 2];
    float3 F = interp_one<P, VEC>(m, ffield, px, py, pz, type[i]);
    const float3 fb = bond_force_one(m, s, x0, bond, (size_t)i, px, py, pz);
    F.x += fb.x;
    F.y += fb.y;
    F.z += fb.z;
    float3 beta = make_float3(0.f, 0.f, 0.f);
    if (s.noise_amp != 0.0f) {
        const float3 z = gauss3(id[i], step_next, s.key0, s.key1);
        beta = make_float3(s.noise_amp * z.x, s.noise_amp * z.y, s.noise_amp * z.z);
    }
    const float p[3] = {px, py, pz};
    const float Fv[3] = {F.x, F.y, F.z};
    const float bv[3] = {beta.x, beta.y, beta.z};
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const float v = w0[3 * (size_t)i + a] + s.half_dt_over_m * Fv[a];
        const float r = p[a] + (s.b_dt * v + s.b_dt2_over_2m * Fv[a] + s.b_dt_over_2m * bv[a]);
        x1[3 * (size_t)i + a] = wrap_pos(r, m.L[a], m.inv_L[a]);
        w1[3 * (size_t)i + a] = s.a_g * (v + s.half_dt_over_m * Fv[a]) + s.b_over_m * bv[a];
    }
}

__global__ void __launch_bounds__(256) axpy_kernel(size_t len, float alpha, const float* __restrict__ f, float* __restrict__ w)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < len) w[i] += alpha * f[i];
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

}  // namespace

static bool can_vectorize(const tild_ctx* c, const float* ffield)
{
    return (c->mesh.N[2] % 4 == 0) && (reinterpret_cast<uintptr_t>(ffield) % 16 == 0) && !(c->prm.flags & TILD_FLAG_NAIVE_INTERP);
}

int launch_interp_force(tild_ctx* c, const float* ffield, const float* x, const int32_t* type, float* f)
{
    const int n = c->mesh.n;
    if (n == 0) return TILD_OK;
    const int nb = (n + 255) / 256;
    const bool vec = can_vectorize(c, ffield);
#define IF(PP)                                                                                          \
    if (vec) interp_force_kernel<PP, true><<<nb, 256, 0, c->stream>>>(c->mesh, ffield, x, type, f);     \
    else interp_force_kernel<PP, false><<<nb, 256, 0, c->stream>>>(c->mesh, ffield, x, type, f)
    switch (c->mesh.P) {
    case 1: IF(1); break;
    case 2: IF(2); break;
    case 3: IF(3); break;
    default: IF(4); break;
    }
#undef IF
    TILD_LAUNCH_CHECK(c, "interp_force_kernel");
    return TILD_OK;
}

int launch_bond_force(tild_ctx* c, const float* x, const int32_t* bond, float* f, bool accumulate)
{
    const int n = c->mesh.n;
    if (n == 0) return TILD_OK;
    bond_force_kernel<<<(n + 255) / 256, 256, 0, c->stream>>>(c->mesh, c->stp, x, bond, f, accumulate ? 1 : 0);
    TILD_LAUNCH_CHECK(c, "bond_force_kernel");
    return TILD_OK;
}

int launch_fused_step(tild_ctx* c)
{
    const int n = c->mesh.n;
    const int a = c->cur;
    // x/w flip between the two buffers; type/id/bond stay in buffer `cur` (they only move on a reorder)
    float* x0 = c->x[a];
    float* w0 = c->w[a];
    float* x1 = c->x[1 - a];
    float* w1 = c->w[1 - a];
    if (n > 0) {
        const int nb = (n + 255) / 256;
        const uint64_t sn = c->step + 1;
        const bool vec = can_vectorize(c, c->ffield);
#define FS(PP)                                                                                                          \
    if (vec) fused_step_kernel<PP, true><<<nb, 256, 0, c->stream>>>(c->mesh, c->stp, sn, c->ffield, x0, w0, c->type[a], c->id[a], c->bond[a], x1, w1); \
    else fused_step_kernel<PP, false><<<nb, 256, 0, c->stream>>>(c->mesh, c->stp, sn, c->ffield, x0, w0, c->type[a], c->id[a], c->bond[a], x1, w1)
        switch (c->mesh.P) {
        case 1: FS(1); break;
        case 2: FS(2); break;
        case 3: FS(3); break;
        default: FS(4); break;
        }
#undef FS
        TILD_LAUNCH_CHECK(c, "fused_step_kernel");
    }
    // swap only the x/w pointers so that `cur` keeps naming the buffer that holds type/id/bond
    c->x[a] = x1;
    c->x[1 - a] = x0;
    c->w[a] = w1;
    c->w[1 - a] = w0;
    return TILD_OK;
}

int launch_make_w(tild_ctx* c, const float* f, float* w, float sign)
{
    const size_t len = 3 * (size_t)c->mesh.n;
    if (len == 0) return TILD_OK;
    axpy_kernel<<<(unsigned)((len + 255) / 256), 256, 0, c->stream>>>(len, sign * c->stp.half_dt_over_m, f, w);
    TILD_LAUNCH_CHECK(c, "axpy_kernel");
    return TILD_OK;
}

int launch_philox_test(tild_ctx* c, const uint32_t* ctr, const uint32_t* key, uint32_t* out, float* gauss, int m)
{
    if (m <= 0) return TILD_OK;
    philox_test_kernel<<<(m + 127) / 128, 128, 0, c->stream>>>(m, ctr, key, out, gauss);
    TILD_LAUNCH_CHECK(c, "philox_test_kernel");
    return TILD_OK;
}
