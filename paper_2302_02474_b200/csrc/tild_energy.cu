// Diagnostics of the current state (not on the timed path): energies and the structure factor.
//   e[0] = kinetic  = m/2 sum |v|^2, v = w + (dt/2m) F (the split-kick state of DESIGN.md "GJF in one pass")
//   e[1] = bonds    = sum_bonds k (|d| - r0)^2, each bond once (Eq. 2)
//   e[2] = non-bonded on the mesh = (1/2V) sum_m u^(k_m) sum_IJ c_IJ Re[n^_I(m) conj(n^_J(m))] (Eq. 3-4 L119-123 with
//          the smeared densities of L139-149; the rho0 shift of Eq. 4 touches m = 0 only and is a constant)
#include "tild_internal.cuh"

namespace {

__device__ __forceinline__ void block_add(double v, double* out)
{
    __shared__ double warp_sum[8];
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
    if ((threadIdx.x & 31) == 0) warp_sum[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int k = 0; k < (int)(blockDim.x >> 5); ++k) s += warp_sum[k];
        atomicAdd(out, s);
    }
}

// half spectrum of the R2C transform: modes with 0 < mz < Nz/2 stand for themselves and their conjugates
template <int S>
__global__ void __launch_bounds__(256) kspace_energy_kernel(KspaceParams k, size_t Mk, const float2* __restrict__ nhat,
                                                            double* __restrict__ out)
{
    double e = 0.0, w = 0.0;
    for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < Mk; idx += (size_t)gridDim.x * blockDim.x) {
        const int mz = (int)(idx % k.Nzc);
        const size_t r = idx / k.Nzc;
        const int my = (int)(r % k.N[1]);
        const int mx = (int)(r / k.N[1]);
        const double u = (double)__ldg(k.ufac[0] + mx) * (double)__ldg(k.ufac[1] + my) * (double)__ldg(k.ufac[2] + mz);  // 1/V inside
        float2 nj[S];
#pragma unroll
        for (int J = 0; J < S; ++J) nj[J] = nhat[(size_t)J * Mk + idx];
        double uel = 0.0;
        if (k.has_el) {
            const double k2 = (double)__ldg(k.k2[0] + mx) + (double)__ldg(k.k2[1] + my) + (double)__ldg(k.k2[2] + mz);
            if (k2 > 0.0) uel = (double)__ldg(k.eel[0] + mx) * (double)__ldg(k.eel[1] + my) * (double)__ldg(k.eel[2] + mz) / k2;
        }
        double acc = 0.0;
#pragma unroll
        for (int I = 0; I < S; ++I)
#pragma unroll
            for (int J = 0; J < S; ++J)
                acc += ((double)k.c[I * TILD_MAX_SPECIES + J] * u + (double)k.qq[I * TILD_MAX_SPECIES + J] * uel) *
                       ((double)nj[I].x * nj[J].x + (double)nj[I].y * nj[J].y);
        const bool self_conjugate = mz == 0 || (k.N[2] % 2 == 0 && mz == k.N[2] / 2);
        e += (self_conjugate ? 0.5 : 1.0) * acc;
        // pressure virial W = -dU/d ln(lambda) of the affine scaling: k -> k / lambda,
        // V -> lambda^3 V, n^ unchanged: every mode contributes its energy times 3 + k . grad_k ln u^, i.e.
        // 3 - sigma2 k^2 for the Gaussian kernel and 3 - 2 k^2 a_q^2 - 2 for the Coulomb kernel (deconvolution: invariant)
        const double k2 = (double)__ldg(k.k2[0] + mx) + (double)__ldg(k.k2[1] + my) + (double)__ldg(k.k2[2] + mz);
        double vacc = 0.0;
#pragma unroll
        for (int I = 0; I < S; ++I)
#pragma unroll
            for (int J = 0; J < S; ++J)
                vacc += ((double)k.c[I * TILD_MAX_SPECIES + J] * u * (3.0 - (double)k.sigma2 * k2) +
                         (double)k.qq[I * TILD_MAX_SPECIES + J] * uel * (1.0 - 2.0 * k2 * (double)k.aq2)) *
                        ((double)nj[I].x * nj[J].x + (double)nj[I].y * nj[J].y);
        w += (self_conjugate ? 0.5 : 1.0) * vacc;
    }
    block_add(e, out + 2);
    __syncthreads();
    block_add(w, out + 4);
}

__global__ void __launch_bounds__(256) particle_energy_kernel(MeshParams m, StepParams s, double mass, const float4* __restrict__ X4,
                                                              const float4* __restrict__ W4, const float4* __restrict__ F4,
                                                              const int32_t* __restrict__ B, double* __restrict__ out)
{
    double ke = 0.0, eb = 0.0, wb = 0.0;
    for (size_t slot = (size_t)blockIdx.x * blockDim.x + threadIdx.x; slot < (size_t)m.n; slot += (size_t)gridDim.x * blockDim.x) {
        const float4 p = X4[slot], w = W4[slot], f = F4[slot];
        const double vx = (double)w.x + (double)s.kick_in * f.x, vy = (double)w.y + (double)s.kick_in * f.y,
                     vz = (double)w.z + (double)s.kick_in * f.z;
        ke += 0.5 * mass * (vx * vx + vy * vy + vz * vz);
        for (int k = 0; k < s.max_bonds; ++k) {
            const int32_t j = B[slot * s.max_bonds + k];
            if (j < 0 || (size_t)j <= slot) continue;            // each bond once: from its lower slot
            const float4 q = X4[j];
            const double dx = min_image(p.x - q.x, m.L[0], m.inv_L[0]), dy = min_image(p.y - q.y, m.L[1], m.inv_L[1]),
                         dz = min_image(p.z - q.z, m.L[2], m.inv_L[2]);
            const double r = sqrt(dx * dx + dy * dy + dz * dz), d = r - (double)s.r0_bond;
            eb += (double)s.k_bond * d * d;
            wb += -2.0 * (double)s.k_bond * d * r;             // bonded virial -dU/dr r (angles are scale invariant)
        }
        if (s.lambda_wlc != 0.0f || s.k_theta != 0.0f) {   // Eq. 16-17, counted by the angle's centre bead
            const int2 bb = *reinterpret_cast<const int2*>(B + 2 * slot);
            if (bb.x >= 0 && bb.y >= 0) {
                const float4 a = X4[bb.x], c = X4[bb.y];
                const float d1[3] = {min_image(a.x - p.x, m.L[0], m.inv_L[0]), min_image(a.y - p.y, m.L[1], m.inv_L[1]),
                                     min_image(a.z - p.z, m.L[2], m.inv_L[2])};
                const float d2[3] = {min_image(c.x - p.x, m.L[0], m.inv_L[0]), min_image(c.y - p.y, m.L[1], m.inv_L[1]),
                                     min_image(c.z - p.z, m.L[2], m.inv_L[2])};
                const double n1 = (double)d1[0] * d1[0] + (double)d1[1] * d1[1] + (double)d1[2] * d1[2];
                const double n2 = (double)d2[0] * d2[0] + (double)d2[1] * d2[1] + (double)d2[2] * d2[2];
                const double dot = (double)d1[0] * d2[0] + (double)d1[1] * d2[1] + (double)d1[2] * d2[2];
                if (n1 > 0.0 && n2 > 0.0) {
                    const double cs = fmin(1.0, fmax(-1.0, dot / sqrt(n1 * n2))), dth = acos(cs) - (double)s.theta0;
                    eb += (double)s.lambda_wlc * (1.0 + cs) + (double)s.k_theta * dth * dth;
                }
            }
        }
    }
    block_add(ke, out + 0);
    __syncthreads();
    block_add(eb, out + 1);
    __syncthreads();
    block_add(wb, out + 3);
}

// S(m) = |sum_{J in mask} n^_J(m)|^2 / N_mask on the half spectrum; N_mask = the m = 0 mode (Eq. 23)
__global__ void __launch_bounds__(256) structure_factor_kernel(int S, uint32_t mask, size_t Mk, const float2* __restrict__ nhat,
                                                               float* __restrict__ sk, int accumulate)
{
    float count = 0.f;
    for (int J = 0; J < S; ++J)
        if (mask >> J & 1u) count += nhat[(size_t)J * Mk].x;
    const float inv = count > 0.f ? 1.0f / count : 0.f;
    for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < Mk; idx += (size_t)gridDim.x * blockDim.x) {
        float re = 0.f, im = 0.f;
        for (int J = 0; J < S; ++J)
            if (mask >> J & 1u) {
                const float2 v = nhat[(size_t)J * Mk + idx];
                re += v.x;
                im += v.y;
            }
        const float v = (re * re + im * im) * inv;
        sk[idx] = accumulate ? sk[idx] + v : v;
    }
}

}  // namespace

int launch_structure_factor(tild_ctx* c, uint32_t mask, float* sk, int accumulate)
{
    structure_factor_kernel<<<592, 256, 0, c->stream>>>(c->mesh.S, mask, c->Mk, c->nhat, sk, accumulate);
    TILD_LAUNCH_CHECK(c, "structure_factor_kernel");
    return TILD_OK;
}

// F4 must hold the total force at the current positions and c->nhat their transformed densities (force_current)
int launch_energy(tild_ctx* c, double* d_out)
{
    TILD_CUDA(c, cudaMemsetAsync(d_out, 0, 5 * sizeof(double), c->stream));   // e[0..2], bonded and mesh virial
    const unsigned nb = 592;
#define KE(SS) case SS: kspace_energy_kernel<SS><<<nb, 256, 0, c->stream>>>(c->ksp, c->Mk, c->nhat, d_out); break;
    switch (c->mesh.S) {
        KE(1) KE(2) KE(3) KE(4) KE(5) KE(6) KE(7) KE(8)
    }
#undef KE
    TILD_LAUNCH_CHECK(c, "kspace_energy_kernel");
    if (c->mesh.n > 0) {
        particle_energy_kernel<<<nb, 256, 0, c->stream>>>(c->mesh, c->stp, c->prm.mass, c->X4[c->cur], c->W4[c->cur], c->F4,
                                                          c->B[c->cur], d_out);
        TILD_LAUNCH_CHECK(c, "particle_energy_kernel");
    }
    return TILD_OK;
}
