// a4: fused k-space kernel.  PAPER.md Eq. 18 L225 with the pair potentials of Eq. 3-4
// L119-123: in Fourier space the convolution "becomes a simple multiplication" (L227):
//   f^_{I,a}(m) = -i k_a(m) u^(k_m) sum_J c_IJ n^_J(m) / V,   u^(k) = exp(-sigma2 |k|^2 / 2)  (L121)
// plus, when a Bjerrum length is set (A22), -i k_a u^_el(k_m) z_I sum_J z_J n^_J(m) / V with the Coulomb kernel
// u^_el(k) = 4 pi l_B exp(-k^2 a_q^2) / k^2 of Gaussian-smeared charges: no extra transform, no extra bandwidth.
// One read of the S transformed densities produces all 3S force spectra.  u^ is separable, so it is three
// 1-D table look-ups (built in double on the host at tild_init; 1/V folded into the x table).
#include "tild_internal.cuh"

#ifndef TILD_XFFT_AHEAD
#define TILD_XFFT_AHEAD 148   // L2 prefetch distance in CTAs (0: off)
#endif

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
// The 3-D transforms are separable.  When Nx = 16, 32, 48, 64, 96, 128, 192 or 256 and S <= 4 the mesh pipeline runs cuFFT only over
// (y, z) -- batched 2-D R2C / C2R over the x planes -- and this kernel does, for 256 / R lines (ky, kz) at a time,
//   forward FFT along x of the S densities -> the multiplication above -> inverse FFT along x of the 3S force spectra,
// in registers (Nx = R1 R2: an R1- and an R2-point transform per line, one shared-memory transpose between them).  Against the
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

// complex add / subtract as one packed fp32 pair instruction (sm_100a FADD2: 384 of them replace 768 FADD in the 16 x 16
// kernel; same rounding; C4 k-space stage 0.1265 -> 0.1251 ms).  TILD_KSPACE_NO_F32X2 builds the scalar form.
__device__ __forceinline__ float2 cadd(float2 a, float2 b)
{
#ifndef TILD_KSPACE_NO_F32X2
    float2 d;
    asm("{.reg .b64 ra, rb, rd;\n mov.b64 ra, {%2, %3};\n mov.b64 rb, {%4, %5};\n add.rn.f32x2 rd, ra, rb;\n mov.b64 {%0, %1}, rd;}"
        : "=f"(d.x), "=f"(d.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));
    return d;
#else
    return make_float2(a.x + b.x, a.y + b.y);
#endif
}
__device__ __forceinline__ float2 csub(float2 a, float2 b)
{
#ifndef TILD_KSPACE_NO_F32X2
    float2 d;
    asm("{.reg .b64 ra, rb, rd;\n mov.b64 ra, {%2, %3};\n mov.b64 rb, {%4, %5};\n sub.rn.f32x2 rd, ra, rb;\n mov.b64 {%0, %1}, rd;}"
        : "=f"(d.x), "=f"(d.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));
    return d;
#else
    return make_float2(a.x - b.x, a.y - b.y);
#endif
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
            v[k] = cadd(e[k], t);
            v[k + R / 2] = csub(e[k], t);
        }
    }
};
template <int SGN>
struct RegFft<1, SGN> {
    static __device__ __forceinline__ void run(float2 (&)[1]) {}
};

// cos / sin of 2 pi j / 24, j = 0 .. 23 (twiddles of the radix-3 splits below)
__host__ __device__ constexpr float cos24q(int j)   // first quadrant, j = 0 .. 6
{
    return j == 0 ? 1.0f : j == 1 ? 0.96592582628906829f : j == 2 ? 0.86602540378443865f : j == 3 ? 0.70710678118654752f
         : j == 4 ? 0.5f : j == 5 ? 0.25881904510252076f : 0.0f;
}
__host__ __device__ constexpr float cos24(int j)
{
    return j <= 6 ? cos24q(j) : j <= 12 ? -cos24q(12 - j) : j <= 18 ? -cos24q(j - 12) : cos24q(24 - j);
}
__host__ __device__ constexpr float sin24(int j) { return cos24((j + 18) % 24); }   // sin x = cos(x - pi/2)

// R = 3 * 2^m points (3, 6, 12, 24): three interleaved power-of-two transforms and a radix-3 butterfly,
//   X[q + (R/3) s] = E0[q] + w3^s W_R^q E1[q] + w3^(2s) W_R^(2q) E2[q],  E_r = DFT of x[3 m + r],  w3 = exp(SGN 2 pi i / 3)
template <int R, int SGN>
struct RegFft3 {
    static __device__ __forceinline__ void run(float2 (&v)[R])
    {
        constexpr int Q = R / 3;
        float2 e[3][Q];
#pragma unroll
        for (int m = 0; m < Q; ++m) {
            e[0][m] = v[3 * m];
            e[1][m] = v[3 * m + 1];
            e[2][m] = v[3 * m + 2];
        }
        RegFft<Q, SGN>::run(e[0]);
        RegFft<Q, SGN>::run(e[1]);
        RegFft<Q, SGN>::run(e[2]);
        constexpr float C3 = -0.5f, S3 = (float)SGN * 0.86602540378443865f;   // w3 = C3 + i S3
#pragma unroll
        for (int q = 0; q < Q; ++q) {
            const float c1 = cos24(q * (24 / R)), s1 = (float)SGN * sin24(q * (24 / R));
            const float c2 = cos24(2 * q * (24 / R)), s2 = (float)SGN * sin24(2 * q * (24 / R));
            const float2 t1 = q == 0 ? e[1][q] : make_float2(c1 * e[1][q].x - s1 * e[1][q].y, c1 * e[1][q].y + s1 * e[1][q].x);
            const float2 t2 = q == 0 ? e[2][q] : make_float2(c2 * e[2][q].x - s2 * e[2][q].y, c2 * e[2][q].y + s2 * e[2][q].x);
            const float2 sum = cadd(t1, t2), dif = csub(t1, t2);
            // E0 + w3 t1 + conj(w3) t2 = E0 + C3 (t1 + t2) + i S3 (t1 - t2); the third output has -S3
            const float2 m = make_float2(e[0][q].x + C3 * sum.x, e[0][q].y + C3 * sum.y);
            const float2 r = make_float2(-S3 * dif.y, S3 * dif.x);
            v[q] = cadd(e[0][q], sum);
            v[q + Q] = cadd(m, r);
            v[q + 2 * Q] = csub(m, r);
        }
    }
};
template <int SGN> struct RegFft<3, SGN> : RegFft3<3, SGN> {};
template <int SGN> struct RegFft<6, SGN> : RegFft3<6, SGN> {};
template <int SGN> struct RegFft<12, SGN> : RegFft3<12, SGN> {};

// One length-N transform per line, N = R1 R2 (R1 <= R2), spread over R2 threads: Cooley-Tukey with the twiddle
// exp(-/+ 2 pi i n2 k1 / N) between an R1-point and an R2-point pass and one shared-memory transpose.
// Forward: thread me (< R2) holds a[j] = in[R2 j + me]; on exit thread me < R1 holds b[j] = out[me + R1 j].
template <int R1, int R2>
__device__ __forceinline__ void line_fft_fwd(float2 (&a)[R1], float2 (&b)[R2], const float2* __restrict__ stw,
                                             float2* __restrict__ ex, int me, int ql)
{
    constexpr int LINES = 256 / R2;
    RegFft<R1, -1>::run(a);
#pragma unroll
    for (int j = 0; j < R1; ++j) {
        const float2 w = stw[me * j];              // exp(-2 pi i me j / N)
        ex[(j * R2 + me) * LINES + ql] = make_float2(a[j].x * w.x - a[j].y * w.y, a[j].x * w.y + a[j].y * w.x);
    }
    __syncthreads();
    if (me < R1) {
#pragma unroll
        for (int j = 0; j < R2; ++j) b[j] = ex[(me * R2 + j) * LINES + ql];
        RegFft<R2, -1>::run(b);
    }
}
// Inverse: thread me < R1 holds b[j] = in[me + R1 j]; on exit thread me (< R2) holds a[j] = out[R2 j + me].
template <int R1, int R2>
__device__ __forceinline__ void line_fft_inv(float2 (&b)[R2], float2 (&a)[R1], const float2* __restrict__ stw,
                                             float2* __restrict__ ex, int me, int ql)
{
    constexpr int LINES = 256 / R2;
    if (me < R1) {
        RegFft<R2, +1>::run(b);
#pragma unroll
        for (int j = 0; j < R2; ++j) {
            const float2 w = stw[me * j];          // conjugated: exp(+2 pi i me j / N)
            ex[(j * R1 + me) * LINES + ql] = make_float2(b[j].x * w.x + b[j].y * w.y, b[j].y * w.x - b[j].x * w.y);
        }
    }
    __syncthreads();
#pragma unroll
    for (int j = 0; j < R1; ++j) a[j] = ex[(me * R1 + j) * LINES + ql];
    RegFft<R1, +1>::run(a);
}

template <int R1, int R2, int S>
__global__ void __launch_bounds__(256, (S <= 2 || R1 <= 8) ? 2 : 1) kspace_xfft_kernel(KspaceParams k, size_t Q, const float2* __restrict__ tw,
                                                             const float2* __restrict__ nhat, float2* __restrict__ fhat)
{
    constexpr int N = R1 * R2, LINES = 256 / R2, EXN = R1 * 256;
    // S >= 3: the transformed densities X of a line live in shared memory (each thread its own S R2 entries), not in registers:
    // 128 registers and two CTAs per SM where the shared memory allows (Nx <= 128), instead of 249 registers and one CTA
    constexpr bool XS = S >= 3;
    constexpr int XSTR = R1 * LINES;    // threads that hold spectra (me < R1)
    extern __shared__ float2 xs[];
    float2* stw = xs;                   // [N] twiddles
    float2* sxu = xs + N;               // [N] (u^_x(m) / V, k_x(m))
    float2* sxe = xs + 2 * N;           // [N] (Coulomb x factor, k_x(m)^2)
    float2* ex = xs + 3 * N;            // [2][R1][R2][LINES], alternating so that one barrier per transpose is enough
    for (int j = threadIdx.x; j < N; j += 256) {
        stw[j] = tw[j];
        sxu[j] = make_float2(__ldg(k.ufac[0] + j), __ldg(k.kgrad[0] + j));
        sxe[j] = make_float2(__ldg(k.eel[0] + j), __ldg(k.k2[0] + j));
    }
    const int ql = threadIdx.x % LINES, me = threadIdx.x / LINES;
    const size_t q = (size_t)blockIdx.x * LINES + ql;
    const bool active = q < Q;
    const size_t qc = active ? q : Q - 1;
    const size_t xstride = (size_t)R2 * Q;          // between the R1 points a thread loads and stores
    int par = 0;

    float2 A[S][R1];
#pragma unroll
    for (int J = 0; J < S; ++J) {
        const float2* src = nhat + ((size_t)J * N + me) * Q + qc;
#pragma unroll
        for (int j = 0; j < R1; ++j) A[J][j] = __ldg(src + (size_t)j * xstride);
    }
#if TILD_XFFT_AHEAD
    {   // the lines of the CTA that follows in this CTA's slot (two CTAs per SM resident) on their way to L2: per species and
        // x one 128-byte piece (LINES consecutive (k_y, k_z) points), S N pieces over 256 threads
        const size_t q0n = ((size_t)blockIdx.x + TILD_XFFT_AHEAD) * LINES;
        if (LINES * sizeof(float2) == 128 && q0n + LINES <= Q)
            for (int i = threadIdx.x; i < S * N; i += 256) asm volatile("prefetch.global.L2 [%0];" ::"l"(nhat + (size_t)i * Q + q0n));
    }
#endif
    const int my = (int)(qc / k.Nzc), mz = (int)(qc % k.Nzc);
    const float uyz = __ldg(k.ufac[1] + my) * __ldg(k.ufac[2] + mz);
    const float ky = __ldg(k.kgrad[1] + my), kz = __ldg(k.kgrad[2] + mz);
    float eyz = 0.f, k2yz = 0.f;
    if (k.has_el) {
        eyz = __ldg(k.eel[1] + my) * __ldg(k.eel[2] + mz);
        k2yz = __ldg(k.k2[1] + my) + __ldg(k.k2[2] + mz);
    }
    __syncthreads();
    float2 X[XS ? 1 : S][R2];                       // threads me < R1: X[J][j] = n^_J(kx = me + R1 j)
    float2* Xs = ex + 2 * EXN + threadIdx.x;        // XS: entry (J, j) of this thread at Xs[(J * R2 + j) * XSTR]
#pragma unroll
    for (int J = 0; J < S; ++J) {
        float2(&Xt)[R2] = X[XS ? 0 : J];
#pragma unroll
        for (int j = 0; j < R2; ++j) Xt[j] = make_float2(0.f, 0.f);
        line_fft_fwd<R1, R2>(A[J], Xt, stw, ex + par * EXN, me, ql);
        par ^= 1;
        if (XS && me < R1) {
#pragma unroll
            for (int j = 0; j < R2; ++j) Xs[(J * R2 + j) * XSTR] = Xt[j];
        }
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
        float2 t[R2];
        if (me < R1) {
#pragma unroll
            for (int j = 0; j < R2; ++j) {
                const int mx = me + R1 * j;
                float gr = 0.f, gi = 0.f;
                float2 xj[S];
#pragma unroll
                for (int J = 0; J < S; ++J) xj[J] = XS ? Xs[(J * R2 + j) * XSTR] : X[XS ? 0 : J][j];
#pragma unroll
                for (int J = 0; J < S; ++J) {
                    gr += cI[J] * xj[J].x;
                    gi += cI[J] * xj[J].y;
                }
                const float2 xu = sxu[mx];
                const float u = xu.x * uyz;
                float tr = u * gr, ti = u * gi;
                if (k.has_el) {
                    float er = 0.f, ei = 0.f;
#pragma unroll
                    for (int J = 0; J < S; ++J) {
                        er += qI[J] * xj[J].x;
                        ei += qI[J] * xj[J].y;
                    }
                    const float2 xe = sxe[mx];
                    const float k2 = xe.y + k2yz;
                    const float uel = k2 > 0.f ? xe.x * eyz / k2 : 0.f;
                    tr += uel * er;
                    ti += uel * ei;
                }
                t[j] = pass == 0 ? make_float2(tr, ti) : make_float2(xu.y * ti, -xu.y * tr);   // pass 1: -i k_x (tr + i ti)
            }
        }
        float2 o[R1];
        line_fft_inv<R1, R2>(t, o, stw, ex + par * EXN, me, ql);
        par ^= 1;
        if (active) {
            if (pass == 0) {
                float2* dy = fhat + (((size_t)I * 3 + 1) * N + me) * Q + q;
                float2* dz = fhat + (((size_t)I * 3 + 2) * N + me) * Q + q;
#pragma unroll
                for (int j = 0; j < R1; ++j) {
                    dy[(size_t)j * xstride] = make_float2(ky * o[j].y, -ky * o[j].x);
                    dz[(size_t)j * xstride] = make_float2(kz * o[j].y, -kz * o[j].x);
                }
            } else {
                float2* dx = fhat + (((size_t)I * 3 + 0) * N + me) * Q + q;
#pragma unroll
                for (int j = 0; j < R1; ++j) dx[(size_t)j * xstride] = o[j];
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

// R2 of the fused x-transform kernel for this mesh (Nx = R1 R2, R1 = Nx / R2 <= R2), 0 when it does not apply
int kspace_xfft_radix(int Nx, int S)
{
    if (S > 4) return 0;   // S = 3, 4: one CTA per SM (the spectra of all species stay in registers)
    return Nx == 256 || Nx == 128 || Nx == 192 || Nx == 96 ? 16 : Nx == 64 || Nx == 32 || Nx == 48 ? 8 : Nx == 16 ? 4 : 0;
}

// dispatch over (Nx, S): OP(R1, R2, S)
#define TILD_XFFT_DISPATCH_S(N_, SS, OP)                                            \
    switch (N_) {                                                                   \
    case 256: OP(16, 16, SS); break;                                                \
    case 192: OP(12, 16, SS); break;                                                \
    case 128: OP(8, 16, SS); break;                                                 \
    case 96: OP(6, 16, SS); break;                                                  \
    case 48: OP(6, 8, SS); break;                                                   \
    case 64: OP(8, 8, SS); break;                                                   \
    case 32: OP(4, 8, SS); break;                                                   \
    default: OP(4, 4, SS); break;                                                   \
    }
#define TILD_XFFT_DISPATCH(N_, S_, OP)                                              \
    do {                                                                            \
        if ((S_) == 1) { TILD_XFFT_DISPATCH_S(N_, 1, OP) }                          \
        else if ((S_) == 2) { TILD_XFFT_DISPATCH_S(N_, 2, OP) }                     \
        else if ((S_) == 3) { TILD_XFFT_DISPATCH_S(N_, 3, OP) }                     \
        else { TILD_XFFT_DISPATCH_S(N_, 4, OP) }                                    \
    } while (0)

// shared memory: 3 tables of N float2 + two transpose buffers of R1 * 256 float2
// + S >= 3: the spectra of the S densities, S R2 entries for each of the R1 * (256 / R2) threads that hold them
static size_t xfft_smem_bytes(int N, int R2, int S)
{
    const size_t xs = S >= 3 ? (size_t)S * R2 * (N / R2) * (256 / R2) : 0;
    return (3 * (size_t)N + 2 * (size_t)(N / R2) * 256 + xs) * sizeof(float2);
}

int tild_kspace_configure(tild_ctx* c)
{
    if (!c->xfft_R) return TILD_OK;
    const int N = c->mesh.N[0];
    const int sm = (int)xfft_smem_bytes(N, c->xfft_R, c->mesh.S);
#define XA(R1_, R2_, SS) TILD_CUDA(c, tild_raise_smem_limit(reinterpret_cast<const void*>(kspace_xfft_kernel<R1_, R2_, SS>), (size_t)sm))
    TILD_XFFT_DISPATCH(N, c->mesh.S, XA);
#undef XA
    return TILD_OK;
}

// nhat: [S][Nx][Ny][Nzc] transformed over (y, z) only; fhat: [S][3][Nx][Ny][Nzc], still to be inverted over (y, z)
int launch_kspace_xfft(tild_ctx* c, const float2* nhat, float2* fhat)
{
    const size_t Q = (size_t)c->mesh.N[1] * c->ksp.Nzc;
    const int N = c->mesh.N[0], lines = 256 / c->xfft_R;
    const unsigned nb = (unsigned)((Q + lines - 1) / lines);
    const size_t sm = xfft_smem_bytes(N, c->xfft_R, c->mesh.S);
#define XL(R1_, R2_, SS) kspace_xfft_kernel<R1_, R2_, SS><<<nb, 256, sm, c->stream>>>(c->ksp, Q, c->xtw, nhat, fhat)
    TILD_XFFT_DISPATCH(N, c->mesh.S, XL);
#undef XL
    TILD_LAUNCH_CHECK(c, "kspace_xfft_kernel");
    return TILD_OK;
}
