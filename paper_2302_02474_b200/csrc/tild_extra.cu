// Extra mesh interactions that ride on the particle-mesh path (SURVEY 8(f) #1 remainder and #4): per-particle charges
// (reading A25) and the Maier-Saupe orientation interaction (PAPER.md IV.D L233-247, Eq. 19-20, reading
// A26).  Both spread a per-particle quantity with the density weights, multiply by a kernel in k-space and interpolate a
// field (and its ik-gradient) back with the same weights.  They write a per-slot force Fext; because the fused
// pass is linear in the force, its effect is added to the outputs of that pass by a small kernel afterwards
// (extra_apply_kernel), so the hot kernels are untouched.  These are not the headline kernels: one thread per particle, global fp32 reductions and gathers, 3-D cuFFT plans.
#include "tild_particle.cuh"

namespace {

constexpr int XT = 256;

// mesh[g] += a_i W(g; r_i) for every slot; a_i from `what`: 0 charge q[id], 1..6 Maier-Saupe component what - 1
__device__ __forceinline__ bool ms_tensor(const MeshParams& m, const float4* __restrict__ X4, const float4* __restrict__ W4,
                                          const int32_t* __restrict__ msp_id, const uint32_t* __restrict__ slot_of_id, size_t slot,
                                          float u[3], float& len, int& partner_slot)
{
    const uint32_t id = __float_as_uint(W4[slot].w);
    const int32_t pj = msp_id[id];
    if (pj < 0) return false;
    partner_slot = (int)slot_of_id[pj];
    const float4 p = X4[slot], q = X4[partner_slot];
    const float d[3] = {min_image(p.x - q.x, m.L[0], m.inv_L[0]), min_image(p.y - q.y, m.L[1], m.inv_L[1]),
                        min_image(p.z - q.z, m.L[2], m.inv_L[2])};
    const float r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
    if (!(r2 > 0.0f)) return false;
    len = sqrtf(r2);
    const float inv = 1.0f / len;
    u[0] = d[0] * inv;
    u[1] = d[1] * inv;
    u[2] = d[2] * inv;
    return true;
}
__device__ __forceinline__ float ms_component(const float u[3], int q)   // xx, yy, zz, xy, xz, yz of u u - I/3
{
    const int A[6] = {0, 1, 2, 0, 0, 1}, Bq[6] = {0, 1, 2, 1, 2, 2};
    return u[A[q]] * u[Bq[q]] - (q < 3 ? (1.0f / 3.0f) : 0.0f);
}

template <int P>
__global__ void __launch_bounds__(XT) extra_spread_kernel(MeshParams m, int what, const float4* __restrict__ X4, const float4* __restrict__ W4,
                                                          const float* __restrict__ q_id, const int32_t* __restrict__ msp_id,
                                                          const uint32_t* __restrict__ slot_of_id, float* __restrict__ mesh)
{
    const size_t slot = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (slot >= (size_t)m.n) return;
    float a;
    if (what == 0) {
        a = q_id[__float_as_uint(W4[slot].w)];
    } else {
        float u[3], len;
        int pj;
        if (!ms_tensor(m, X4, W4, msp_id, slot_of_id, slot, u, len, pj)) return;
        a = ms_component(u, what - 1);
    }
    if (a == 0.0f) return;
    int b[3];
    float w[3][P];
    index_weights<P>(m, X4[slot], b, w);
#pragma unroll
    for (int jx = 0; jx < P; ++jx) {
        const size_t ox = (size_t)wrap_idx(b[0] + jx, m.N[0]) * m.N[1];
#pragma unroll
        for (int jy = 0; jy < P; ++jy) {
            const size_t row = (ox + wrap_idx(b[1] + jy, m.N[1])) * m.N[2];
            const float wxy = a * w[0][jx] * w[1][jy];
#pragma unroll
            for (int jz = 0; jz < P; ++jz) atomicAdd(mesh + row + wrap_idx(b[2] + jz, m.N[2]), wxy * w[2][jz]);
        }
    }
}

// spectra of the fields to interpolate.  in: rho^ (half spectrum).  mode 0 (charges): out[a] = -i k_a u^_el rho^ / V, a = 0..2.
// mode 1 (Maier-Saupe): out[0] = u^ rho^ / V (Phi^), out[1 + a] = i k_a u^ rho^ / V (its gradient).
__global__ void __launch_bounds__(XT) extra_kspace_kernel(KspaceParams k, size_t Mk, int mode, const float2* __restrict__ in,
                                                          float2* __restrict__ out)
{
    const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= Mk) return;
    const int mz = (int)(idx % k.Nzc);
    const size_t r = idx / k.Nzc;
    const int my = (int)(r % k.N[1]), mx = (int)(r / k.N[1]);
    const float kg[3] = {__ldg(k.kgrad[0] + mx), __ldg(k.kgrad[1] + my), __ldg(k.kgrad[2] + mz)};
    const float2 v = in[idx];
    if (mode == 0) {
        const float k2 = __ldg(k.k2[0] + mx) + __ldg(k.k2[1] + my) + __ldg(k.k2[2] + mz);
        const float uel = k2 > 0.f ? __ldg(k.eel[0] + mx) * __ldg(k.eel[1] + my) * __ldg(k.eel[2] + mz) / k2 : 0.f;   // 4 pi l_B / V inside
#pragma unroll
        for (int a = 0; a < 3; ++a) out[(size_t)a * Mk + idx] = make_float2(kg[a] * uel * v.y, -kg[a] * uel * v.x);
    } else {
        const float u = __ldg(k.ufac[0] + mx) * __ldg(k.ufac[1] + my) * __ldg(k.ufac[2] + mz);                          // 1 / V inside
        out[idx] = make_float2(u * v.x, u * v.y);
#pragma unroll
        for (int a = 0; a < 3; ++a) out[(size_t)(1 + a) * Mk + idx] = make_float2(-kg[a] * u * v.y, kg[a] * u * v.x);
    }
}

template <int P>
__device__ __forceinline__ void gather_fields(const MeshParams& m, const float4& p, const float* __restrict__ f, int nf, float out[4])
{
    int b[3];
    float w[3][P];
    index_weights<P>(m, p, b, w);
    for (int c = 0; c < nf; ++c) out[c] = 0.f;
#pragma unroll
    for (int jx = 0; jx < P; ++jx) {
        const size_t ox = (size_t)wrap_idx(b[0] + jx, m.N[0]) * m.N[1];
#pragma unroll
        for (int jy = 0; jy < P; ++jy) {
            const size_t row = (ox + wrap_idx(b[1] + jy, m.N[1])) * m.N[2];
            const float wxy = w[0][jx] * w[1][jy];
#pragma unroll
            for (int jz = 0; jz < P; ++jz) {
                const size_t g = row + wrap_idx(b[2] + jz, m.N[2]);
                const float ww = wxy * w[2][jz];
                for (int c = 0; c < nf; ++c) out[c] += ww * __ldg(f + (size_t)c * m.M + g);
            }
        }
    }
}

// what == 0: Fext[slot] += q E(r);  what = 1..6: Fext += 2 pref mult S_q grad Phi_q(r), acc += Phi_q contributions to Phi u
template <int P>
__global__ void __launch_bounds__(XT) extra_gather_kernel(MeshParams m, int what, float pref, const float* __restrict__ fields,
                                                          const float4* __restrict__ X4, const float4* __restrict__ W4,
                                                          const float* __restrict__ q_id, const int32_t* __restrict__ msp_id,
                                                          const uint32_t* __restrict__ slot_of_id, float4* __restrict__ Fext,
                                                          float4* __restrict__ acc)
{
    const size_t slot = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (slot >= (size_t)m.n) return;
    float val[4];
    if (what == 0) {
        const float q = q_id[__float_as_uint(W4[slot].w)];
        if (q == 0.0f) return;
        gather_fields<P>(m, X4[slot], fields, 3, val);
        float4 f = Fext[slot];
        f.x += q * val[0];
        f.y += q * val[1];
        f.z += q * val[2];
        Fext[slot] = f;
        return;
    }
    float u[3], len;
    int pj;
    if (!ms_tensor(m, X4, W4, msp_id, slot_of_id, slot, u, len, pj)) return;
    gather_fields<P>(m, X4[slot], fields, 4, val);
    const int qc = what - 1;
    const int A[6] = {0, 1, 2, 0, 0, 1}, Bq[6] = {0, 1, 2, 1, 2, 2};
    const float sq = ms_component(u, qc) * (qc < 3 ? 1.0f : 2.0f) * 2.0f * pref;     // S_i : d_a Phi, off-diagonals twice
    float4 f = Fext[slot];
    f.x += sq * val[1];
    f.y += sq * val[2];
    f.z += sq * val[3];
    Fext[slot] = f;
    float4 pu = acc[slot];                                                           // (Phi u)_a = sum_b Phi_ab u_b
    float puv[3] = {pu.x, pu.y, pu.z};
    puv[A[qc]] += val[0] * u[Bq[qc]];
    if (qc >= 3) puv[Bq[qc]] += val[0] * u[A[qc]];
    acc[slot] = make_float4(puv[0], puv[1], puv[2], 0.f);
}

// orientation part: G = 4 pref (I - u u) Phi u / |d| on the centre, -G on its partner
__global__ void __launch_bounds__(XT) ms_orient_kernel(MeshParams m, float pref, const float4* __restrict__ X4, const float4* __restrict__ W4,
                                                       const int32_t* __restrict__ msp_id, const uint32_t* __restrict__ slot_of_id,
                                                       const float4* __restrict__ acc, float4* __restrict__ Fext)
{
    const size_t slot = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (slot >= (size_t)m.n) return;
    float u[3], len;
    int pj;
    if (!ms_tensor(m, X4, W4, msp_id, slot_of_id, slot, u, len, pj)) return;
    const float4 pu = acc[slot];
    const float upu = u[0] * pu.x + u[1] * pu.y + u[2] * pu.z, sc = 4.0f * pref / len;
    const float G[3] = {sc * (pu.x - u[0] * upu), sc * (pu.y - u[1] * upu), sc * (pu.z - u[2] * upu)};
    float* fi = reinterpret_cast<float*>(Fext + slot);
    float* fj = reinterpret_cast<float*>(Fext + pj);
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        atomicAdd(fi + a, G[a]);
        atomicAdd(fj + a, -G[a]);
    }
}

// The fused pass is linear in the force: r' = r + b_dt v + b_dt2_over_2m F + ..., w' = a_g (v + w_fr F) + ..., v = w + kick_in F.
// An extra force dF therefore moves its outputs by dr = (b_dt kick_in + b_dt2_over_2m) dF and dw' = a_g (kick_in + w_fr) dF
// (Euler-Maruyama: dr = (dt/gamma) dF), which this kernel applies after the pass -- the hot kernels carry no branch for it.
__global__ void __launch_bounds__(XT) extra_apply_kernel(MeshParams m, StepParams s, int mode, float kick_in, const float4* __restrict__ Fext,
                                                         float4* __restrict__ F4, float4* __restrict__ X4o, float4* __restrict__ W4o)
{
    const size_t slot = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (slot >= (size_t)m.n) return;
    float4 e = Fext[slot];
    if (s.dim2) e.z = 0.0f;
    if (mode == 1) {
        float4 f = F4[slot];
        f.x += e.x;
        f.y += e.y;
        f.z += e.z;
        F4[slot] = f;
        return;
    }
    const bool em = s.integrator == TILD_INTEGRATOR_EM;
    const float cr = em ? s.em_drift : s.b_dt * kick_in + s.b_dt2_over_2m;
    float4 x = X4o[slot];
    x.x = wrap_pos(x.x + cr * e.x, m.L[0], m.inv_L[0]);
    x.y = wrap_pos(x.y + cr * e.y, m.L[1], m.inv_L[1]);
    if (!s.dim2) x.z = wrap_pos(x.z + cr * e.z, m.L[2], m.inv_L[2]);
    X4o[slot] = x;
    if (!em) {
        const float cw = s.a_g * (kick_in + s.w_fr);
        float4 w = W4o[slot];
        w.x += cw * e.x;
        w.y += cw * e.y;
        w.z += cw * e.z;
        W4o[slot] = w;
    }
}

__global__ void __launch_bounds__(XT) slot_of_id_kernel(int n, const float4* __restrict__ W4, uint32_t* __restrict__ slot_of_id)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s < n) slot_of_id[__float_as_uint(W4[s].w)] = (uint32_t)s;
}

}  // namespace

#define TILD_XFFT(c, call)                                                                 \
    do {                                                                                   \
        cufftResult r__ = (call);                                                          \
        if (r__ != CUFFT_SUCCESS) return tild_fail((c), TILD_ECUFFT, "%s: cufft error %d", #call, (int)r__); \
    } while (0)

int launch_slot_of_id(tild_ctx* c)
{
    const int n = c->mesh.n;
    if (n == 0 || !c->slot_of_id) return TILD_OK;
    slot_of_id_kernel<<<(n + XT - 1) / XT, XT, 0, c->stream>>>(n, c->W4[c->cur], c->slot_of_id);
    TILD_LAUNCH_CHECK(c, "slot_of_id_kernel");
    return TILD_OK;
}

template <int P>
static int extra_forces_p(tild_ctx* c, const float4* X4, const float4* W4)
{
    const int n = c->mesh.n;
    const unsigned nb = (unsigned)((n + XT - 1) / XT), nbk = (unsigned)((c->Mk + XT - 1) / XT);
    const size_t M = c->M, Mk = c->Mk;
    cufftComplex* xh = reinterpret_cast<cufftComplex*>(c->xh);
    TILD_CUDA(c, cudaMemsetAsync(c->Fext, 0, sizeof(float4) * (size_t)n, c->stream));
    if (c->has_q && c->prm.bjerrum > 0.0) {
        TILD_CUDA(c, cudaMemsetAsync(c->xr, 0, sizeof(float) * M, c->stream));
        extra_spread_kernel<P><<<nb, XT, 0, c->stream>>>(c->mesh, 0, X4, W4, c->q_id, c->msp_id, c->slot_of_id, c->xr);
        TILD_LAUNCH_CHECK(c, "extra_spread_kernel");
        TILD_XFFT(c, cufftExecR2C(c->plan_x_r2c, c->xr, xh));
        extra_kspace_kernel<<<nbk, XT, 0, c->stream>>>(c->ksp, Mk, 0, c->xh, c->xh + Mk);
        TILD_LAUNCH_CHECK(c, "extra_kspace_kernel");
        for (int a = 0; a < 3; ++a) TILD_XFFT(c, cufftExecC2R(c->plan_x_c2r, xh + (size_t)(1 + a) * Mk, c->xr + (size_t)a * M));
        extra_gather_kernel<P><<<nb, XT, 0, c->stream>>>(c->mesh, 0, 0.f, c->xr, X4, W4, c->q_id, c->msp_id, c->slot_of_id, c->Fext, c->xacc);
        TILD_LAUNCH_CHECK(c, "extra_gather_kernel");
    }
    if (c->has_ms && c->prm.mu_ms != 0.0) {
        const float pref = (float)(c->prm.mu_ms / c->rho0);
        TILD_CUDA(c, cudaMemsetAsync(c->xacc, 0, sizeof(float4) * (size_t)n, c->stream));
        for (int q = 0; q < 6; ++q) {
            TILD_CUDA(c, cudaMemsetAsync(c->xr, 0, sizeof(float) * M, c->stream));
            extra_spread_kernel<P><<<nb, XT, 0, c->stream>>>(c->mesh, 1 + q, X4, W4, c->q_id, c->msp_id, c->slot_of_id, c->xr);
            TILD_LAUNCH_CHECK(c, "extra_spread_kernel");
            TILD_XFFT(c, cufftExecR2C(c->plan_x_r2c, c->xr, xh));
            extra_kspace_kernel<<<nbk, XT, 0, c->stream>>>(c->ksp, Mk, 1, c->xh, c->xh + Mk);
            TILD_LAUNCH_CHECK(c, "extra_kspace_kernel");
            for (int a = 0; a < 4; ++a) TILD_XFFT(c, cufftExecC2R(c->plan_x_c2r, xh + (size_t)(1 + a) * Mk, c->xr + (size_t)a * M));
            extra_gather_kernel<P><<<nb, XT, 0, c->stream>>>(c->mesh, 1 + q, pref, c->xr, X4, W4, c->q_id, c->msp_id, c->slot_of_id, c->Fext, c->xacc);
            TILD_LAUNCH_CHECK(c, "extra_gather_kernel");
        }
        ms_orient_kernel<<<nb, XT, 0, c->stream>>>(c->mesh, pref, X4, W4, c->msp_id, c->slot_of_id, c->xacc, c->Fext);
        TILD_LAUNCH_CHECK(c, "ms_orient_kernel");
    }
    return TILD_OK;
}

// Fext[slot] = force of the extra mesh interactions at the positions X4 (slot order W4)
int launch_extra_forces(tild_ctx* c, const float4* X4, const float4* W4)
{
    const bool active = c->Fext && ((c->has_q && c->prm.bjerrum > 0.0) || (c->has_ms && c->prm.mu_ms != 0.0));
    c->x_active = active && c->mesh.n > 0;
    if (!c->x_active) return TILD_OK;
    switch (c->mesh.P) {
    case 1: return extra_forces_p<1>(c, X4, W4);
    case 2: return extra_forces_p<2>(c, X4, W4);
    case 3: return extra_forces_p<3>(c, X4, W4);
    case 4: return extra_forces_p<4>(c, X4, W4);
    default: return extra_forces_p<5>(c, X4, W4);
    }
}

int launch_extra_apply(tild_ctx* c, int mode, float kick_in, float4* X4o, float4* W4o)
{
    if (!c->x_active) return TILD_OK;
    const int n = c->mesh.n;
    extra_apply_kernel<<<(n + XT - 1) / XT, XT, 0, c->stream>>>(c->mesh, c->stp, mode, kick_in, c->Fext, c->F4, X4o, W4o);
    TILD_LAUNCH_CHECK(c, "extra_apply_kernel");
    return TILD_OK;
}
