// a4: fused k-space kernel.  PAPER.md Eq. 18 L225 with the pair potentials of Eq. 3-4
// L119-123: in Fourier space the convolution "becomes a simple multiplication" (L227):
//   f^_{I,a}(m) = -i k_a(m) u^(k_m) sum_J c_IJ n^_J(m) / V,   u^(k) = exp(-sigma2 |k|^2 / 2)  (L121)
// plus, when a Bjerrum length is set (A22), -i k_a u^_el(k_m) z_I sum_J z_J n^_J(m) / V with the Coulomb kernel
// u^_el(k) = 4 pi l_B exp(-k^2 a_q^2) / k^2 of Gaussian-smeared charges: no extra transform, no extra bandwidth.
// One read of the S transformed densities produces all 3S force spectra.  u^ is separable, so it is three
// 1-D table look-ups (built in double on the host at tild_init; 1/V folded into the x table).
#include "tild_internal.cuh"

namespace {

template <int S>
__global__ void __launch_bounds__(256) kspace_kernel(KspaceParams k, size_t Mk, const float2* __restrict__ nhat,
                                                     float2* __restrict__ fhat)
{
    const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= Mk) return;
    const int mz = (int)(idx % k.Nzc);
    const size_t r = idx / k.Nzc;
    const int my = (int)(r % k.N[1]);
    const int mx = (int)(r / k.N[1]);
    const float u = __ldg(k.ufac[0] + mx) * __ldg(k.ufac[1] + my) * __ldg(k.ufac[2] + mz);
    const float kx = __ldg(k.kgrad[0] + mx), ky = __ldg(k.kgrad[1] + my), kz = __ldg(k.kgrad[2] + mz);
    float uel = 0.f;
    if (k.has_el) {   // Coulomb kernel between Gaussian-smeared unit charges (A22); the k = 0 mode is dropped
        const float k2 = __ldg(k.k2[0] + mx) + __ldg(k.k2[1] + my) + __ldg(k.k2[2] + mz);
        uel = k2 > 0.f ? __ldg(k.eel[0] + mx) * __ldg(k.eel[1] + my) * __ldg(k.eel[2] + mz) / k2 : 0.f;
    }
    float2 nj[S];
#pragma unroll
    for (int J = 0; J < S; ++J) nj[J] = nhat[(size_t)J * Mk + idx];
#pragma unroll
    for (int I = 0; I < S; ++I) {
        float gr = 0.f, gi = 0.f, er = 0.f, ei = 0.f;
#pragma unroll
        for (int J = 0; J < S; ++J) {
            const float cij = k.c[I * TILD_MAX_SPECIES + J];
            gr += cij * nj[J].x;
            gi += cij * nj[J].y;
            if (k.has_el) {
                const float q = k.qq[I * TILD_MAX_SPECIES + J];
                er += q * nj[J].x;
                ei += q * nj[J].y;
            }
        }
        const float tr = u * gr + uel * er, ti = u * gi + uel * ei;
        // -i k (tr + i ti) = k ti - i k tr
        fhat[((size_t)I * 3 + 0) * Mk + idx] = make_float2(kx * ti, -kx * tr);
        fhat[((size_t)I * 3 + 1) * Mk + idx] = make_float2(ky * ti, -ky * tr);
        fhat[((size_t)I * 3 + 2) * Mk + idx] = make_float2(kz * ti, -kz * tr);
    }
}

}  // namespace

int launch_kspace(tild_ctx* c, const float2* nhat, float2* fhat)
{
    const size_t Mk = c->Mk;
    const unsigned nb = (unsigned)((Mk + 255) / 256);
#define KS(SS) case SS: kspace_kernel<SS><<<nb, 256, 0, c->stream>>>(c->ksp, Mk, nhat, fhat); break;
    switch (c->mesh.S) {
        KS(1) KS(2) KS(3) KS(4) KS(5) KS(6) KS(7) KS(8)
    }
#undef KS
    TILD_LAUNCH_CHECK(c, "kspace_kernel");
    return TILD_OK;
}
