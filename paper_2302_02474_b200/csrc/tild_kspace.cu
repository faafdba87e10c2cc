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


// ---- fused x-transform variant --------------------------------------------------------------------------------------
// The 3-D transforms are separable.  When Nx = R^2 (R = 4, 8, 16) and S <= 2 the mesh pipeline runs cuFFT only over
// (y, z) -- batched 2-D R2C / C2R over the x planes -- and this kernel does, for 256 / R lines (ky, kz) at a time,
//   forward FFT along x of the S densities -> the multiplication above -> inverse FFT along x of the 3S force spectra,
// in registers (two R-point transforms per length-N transform, one shared-memory transpose between them).  Against the
// 3-D plans this drops the x passes of all 4S transforms and the round trip of n^ and f^ through HBM between them:
// the stage still reads S and writes 3S half-spectra (its algorithmic bytes), nothing else.  Since k_y and k_z are
// constant along a line, only IFFT_x(t) and IFFT_x(-i k_x t) are computed; the y and z components scale the former.
__host__ __device__ constexpr float cos16(int j)
{
    return j == 0 ? 1.0f : j == 1 ? 0.92387953251128674f : j == 2 ? 0.70710678118654752f : j == 3 ? 0.38268343236508977f
         : j == 4 ? 0.0f : j == 5 ? -0.38268343236508977f : j == 6 ? -0.70710678118654752f : -0.92387953251128674f;
}
__host__ __device__ constexpr float sin16(int j)
{
    return j == 0 ? 0.0f : j == 1 ? 0.38268343236508977f : j == 2 ? 0.70710678118654752f : j == 3 ? 0.92387953251128674f
         : j == 4 ? 1.0f : j == 5 ? 0.92387953251128674f : j == 6 ? 0.70710678118654752f : 0.38268343236508977f;
}

// R-point DFT on registers, decimation in time: v[k] <- sum_n v[n] exp(SGN 2 pi i n k / R)
template <int R, int SGN>
struct RegFft {
    static __device__ __forceinline__ void run(float2 (&v)[R])
    {
        float2 e[R / 2], o[R / 2];
#pragma unroll
        for (int k = 0; k < R / 2; ++k) {
            e[k] = v[2 * k];
            o[k] = v[2 * k + 1];
        }
        RegFft<R / 2, SGN>::run(e);
        RegFft<R / 2, SGN>::run(o);
#pragma unroll
        for (int k = 0; k < R / 2; ++k) {
            float2 t;
            if (k == 0) {
                t = o[k];
            } else if (4 * k == R) {           // w = SGN i
                t = make_float2(-(float)SGN * o[k].y, (float)SGN * o[k].x);
            } else {
                const float wr = cos16(k * (16 / R)), wi = (float)SGN * sin16(k * (16 / R));
                t = make_float2(wr * o[k].x - wi * o[k].y, wr * o[k].y + wi * o[k].x);
            }
            v[k] = make_float2(e[k].x + t.x, e[k].y + t.y);
            v[k + R / 2] = make_float2(e[k].x - t.x, e[k].y - t.y);
        }
    }
};
template <int SGN>
struct RegFft<1, SGN> {
    static __device__ __forceinline__ void run(float2 (&)[1]) {}
};

// One length-N (N = R^2) transform per line, spread over R threads.  On entry thread `me` of a line holds
// v[j] = in[R j + me] (forward) or in[me + R j] (inverse); on exit out[me + R j] (forward) or out[R j + me] (inverse):
// N = R^2 Cooley-Tukey with the twiddle exp(SGN 2 pi i me k / N) between the two R-point passes.
template <int R, int SGN>
__device__ __forceinline__ void line_fft(float2 (&v)[R], const float2* __restrict__ stw, float2* __restrict__ ex, int me, int ql)
{
    constexpr int LINES = 256 / R;
    RegFft<R, SGN>::run(v);
#pragma unroll
    for (int j = 0; j < R; ++j) {
        const float2 w = stw[me * j];              // exp(-2 pi i me j / N); conjugated for the inverse
        const float wi = SGN < 0 ? w.y : -w.y;
        ex[(j * R + me) * LINES + ql] = make_float2(v[j].x * w.x - v[j].y * wi, v[j].x * wi + v[j].y * w.x);
    }
    __syncthreads();
#pragma unroll
    for (int j = 0; j < R; ++j) v[j] = ex[(me * R + j) * LINES + ql];
    RegFft<R, SGN>::run(v);
}

template <int R, int S>
__global__ void __launch_bounds__(256, 2) kspace_xfft_kernel(KspaceParams k, size_t Q, const float2* __restrict__ tw,
                                                             const float2* __restrict__ nhat, float2* __restrict__ fhat)
{
    constexpr int N = R * R, LINES = 256 / R, EXN = R * 256;
    extern __shared__ float2 xs[];
    float2* stw = xs;                   // [N] twiddles
    float2* sxu = xs + N;               // [N] (u^_x(m) / V, k_x(m))
    float2* sxe = xs + 2 * N;           // [N] (Coulomb x factor, k_x(m)^2)
    float2* ex = xs + 3 * N;            // [2][R][R][LINES], alternating so that one barrier per transpose is enough
    for (int j = threadIdx.x; j < N; j += 256) {
        stw[j] = tw[j];
        sxu[j] = make_float2(__ldg(k.ufac[0] + j), __ldg(k.kgrad[0] + j));
        sxe[j] = make_float2(__ldg(k.eel[0] + j), __ldg(k.k2[0] + j));
    }
    const int ql = threadIdx.x % LINES, me = threadIdx.x / LINES;
    const size_t q = (size_t)blockIdx.x * LINES + ql;
    const bool active = q < Q;
    const size_t qc = active ? q : Q - 1;
    const size_t xstride = (size_t)R * Q;           // between the R points a thread holds
    int par = 0;

    float2 X[S][R];                                 // X[J][j] = n^_J(kx = me + R j) after the forward transform
#pragma unroll
    for (int J = 0; J < S; ++J) {
        const float2* src = nhat + ((size_t)J * N + me) * Q + qc;
#pragma unroll
        for (int j = 0; j < R; ++j) X[J][j] = __ldg(src + (size_t)j * xstride);
    }
    const int my = (int)(qc / k.Nzc), mz = (int)(qc % k.Nzc);
    const float uyz = __ldg(k.ufac[1] + my) * __ldg(k.ufac[2] + mz);
    const float ky = __ldg(k.kgrad[1] + my), kz = __ldg(k.kgrad[2] + mz);
    float eyz = 0.f, k2yz = 0.f;
    if (k.has_el) {
        eyz = __ldg(k.eel[1] + my) * __ldg(k.eel[2] + mz);
        k2yz = __ldg(k.k2[1] + my) + __ldg(k.k2[2] + mz);
    }
    __syncthreads();
#pragma unroll
    for (int J = 0; J < S; ++J) {
        line_fft<R, -1>(X[J], stw, ex + par * EXN, me, ql);
        par ^= 1;
    }
    // 2S inverse transforms: (I, pass) with pass 0: t_I -> y and z components, pass 1: -i k_x t_I -> x component
#pragma unroll 1
    for (int ip = 0; ip < 2 * S; ++ip) {
        const int I = ip >> 1, pass = ip & 1;
        float cI[S], qI[S];
#pragma unroll
        for (int J = 0; J < S; ++J) {
            cI[J] = k.c[I * TILD_MAX_SPECIES + J];
            qI[J] = k.qq[I * TILD_MAX_SPECIES + J];
        }
        float2 t[R];
#pragma unroll
        for (int j = 0; j < R; ++j) {
            const int mx = me + R * j;
            float gr = 0.f, gi = 0.f;
#pragma unroll
            for (int J = 0; J < S; ++J) {
                gr += cI[J] * X[J][j].x;
                gi += cI[J] * X[J][j].y;
            }
            const float2 xu = sxu[mx];
            const float u = xu.x * uyz;
            float tr = u * gr, ti = u * gi;
            if (k.has_el) {
                float er = 0.f, ei = 0.f;
#pragma unroll
                for (int J = 0; J < S; ++J) {
                    er += qI[J] * X[J][j].x;
                    ei += qI[J] * X[J][j].y;
                }
                const float2 xe = sxe[mx];
                const float k2 = xe.y + k2yz;
                const float uel = k2 > 0.f ? xe.x * eyz / k2 : 0.f;
                tr += uel * er;
                ti += uel * ei;
            }
            t[j] = pass == 0 ? make_float2(tr, ti) : make_float2(xu.y * ti, -xu.y * tr);   // pass 1: -i k_x (tr + i ti)
        }
        line_fft<R, +1>(t, stw, ex + par * EXN, me, ql);
        par ^= 1;
        if (active) {
            if (pass == 0) {
                float2* dy = fhat + (((size_t)I * 3 + 1) * N + me) * Q + q;
                float2* dz = fhat + (((size_t)I * 3 + 2) * N + me) * Q + q;
#pragma unroll
                for (int j = 0; j < R; ++j) {
                    dy[(size_t)j * xstride] = make_float2(ky * t[j].y, -ky * t[j].x);
                    dz[(size_t)j * xstride] = make_float2(kz * t[j].y, -kz * t[j].x);
                }
            } else {
                float2* dx = fhat + (((size_t)I * 3 + 0) * N + me) * Q + q;
#pragma unroll
                for (int j = 0; j < R; ++j) dx[(size_t)j * xstride] = t[j];
            }
        }
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

// the radix R of the fused x-transform kernel for this mesh, 0 when it does not apply
int kspace_xfft_radix(int Nx, int S)
{
    if (S > 2) return 0;
    return Nx == 256 ? 16 : Nx == 64 ? 8 : Nx == 16 ? 4 : 0;
}

size_t kspace_xfft_smem(int R) { return (3 * (size_t)R * R + 2 * (size_t)R * 256) * sizeof(float2); }

int tild_kspace_configure(tild_ctx* c)
{
    if (!c->xfft_R) return TILD_OK;
    const int sm = (int)kspace_xfft_smem(c->xfft_R);
#define XA(RR, SS) TILD_CUDA(c, cudaFuncSetAttribute(kspace_xfft_kernel<RR, SS>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm))
    if (c->mesh.S == 1) {
        if (c->xfft_R == 16) XA(16, 1); else if (c->xfft_R == 8) XA(8, 1); else XA(4, 1);
    } else {
        if (c->xfft_R == 16) XA(16, 2); else if (c->xfft_R == 8) XA(8, 2); else XA(4, 2);
    }
#undef XA
    return TILD_OK;
}

// nhat: [S][Nx][Ny][Nzc] transformed over (y, z) only; fhat: [S][3][Nx][Ny][Nzc], still to be inverted over (y, z)
int launch_kspace_xfft(tild_ctx* c, const float2* nhat, float2* fhat)
{
    const size_t Q = (size_t)c->mesh.N[1] * c->ksp.Nzc;
    const int R = c->xfft_R, lines = 256 / R;
    const unsigned nb = (unsigned)((Q + lines - 1) / lines);
    const size_t sm = kspace_xfft_smem(R);
#define XL(RR, SS) kspace_xfft_kernel<RR, SS><<<nb, 256, sm, c->stream>>>(c->ksp, Q, c->xtw, nhat, fhat)
    if (c->mesh.S == 1) {
        if (R == 16) XL(16, 1); else if (R == 8) XL(8, 1); else XL(4, 1);
    } else {
        if (R == 16) XL(16, 2); else if (R == 8) XL(8, 2); else XL(4, 2);
    }
#undef XL
    TILD_LAUNCH_CHECK(c, "kspace_xfft_kernel");
    return TILD_OK;
}
