// Internal declarations of libtild (sm_100a).  Not part of the C-ABI; see include/tild.h.
#pragma once
#include <cuda_runtime.h>
#include <cufft.h>
#include <stdint.h>

#include "../../include/tild.h"

#define TILD_MAX_TIMED_STEPS 128
#define TILD_N_STAGE_EVENTS 8  // start, after sort, spread, fft_fwd, kspace, fft_inv, interp, (spare)

// ---- kernel parameter blocks (passed by value) -------------------------------------------------
struct MeshParams {
    int n, S, P;
    int N[3];
    float inv_h[3];  // fl32(N/L): the canonical fp32 index-map scale (A15)
    float L[3];
    float inv_L[3];
    long long M;     // Nx*Ny*Nz
};

// Tiling of the cell grid for the shared-memory spread (tild_spread.cu) and the tile-major particle order.
struct TileParams {
    int T[3];       // tile edge in cells (clipped to the grid)
    int nt[3];      // tiles per axis = ceil(N/T)
    int E[3];       // shared tile edge in nodes = T + stencil halo + 2*margin
    int lo;         // nodes below the tile's first cell held in shared memory (low halo + margin)
    int TV;         // T[0]*T[1]*T[2]: cells per tile; sort key = (tile*S + species)*TV + local cell
    int ntiles;
    unsigned nbins; // ntiles*S*TV
    size_t smem_bytes;
    int enabled;    // 0: grid too small for the tile kernel (any N < 8) -> per-particle spread
};

struct KspaceParams {
    int S;
    int N[3];
    int Nzc;                 // Nz/2 + 1
    const float* kgrad[3];   // k_a(m), 0 at the Nyquist index of even N (A6)
    const float* ufac[3];    // exp(-sigma2 k_a(m)^2 / 2); ufac[0] also carries 1/V
    float c[TILD_MAX_SPECIES * TILD_MAX_SPECIES];  // c_IJ (1/V folded into ufac[0])
};

struct StepParams {
    float half_dt_over_m;  // dt/2m
    float a_g;             // (1 - gamma dt/2m)/(1 + gamma dt/2m)
    float b_dt;            // b dt
    float b_dt2_over_2m;   // b dt^2/2m
    float b_dt_over_2m;    // b dt/2m
    float b_over_m;        // b/m
    float noise_amp;       // sqrt(2 gamma kT dt); 0 disables the draw
    float k_bond, r0_bond;
    int max_bonds;
    uint32_t key0, key1;   // Philox key = seed lo, hi
};

// ---- context -----------------------------------------------------------------------------------
struct tild_ctx {
    tild_params prm;
    cudaStream_t stream;
    MeshParams mesh;
    KspaceParams ksp;
    StepParams stp;
    size_t M, Mk;
    TileParams tile;
    size_t max_bins;      // max(M, tile.nbins)

    // carved from the caller's workspace
    float* x[2];
    float* w[2];
    int32_t* type[2];
    uint32_t* id[2];
    int32_t* bond[2];
    int cur;
    float* grid;        // [S][M]
    float2* nhat;       // [S][Mk]
    float2* fhat;       // [3S][Mk]
    float* ffield;      // [3S][M]
    float* fpart;       // [n][3] scratch forces (internal order)
    uint32_t* key;      // [n]
    uint32_t* perm;     // [n]
    uint32_t* tile_start;  // [tile.nbins+1] tile-major cell offsets of the internal (sorted) state
    uint32_t* cell_start;  // [max_bins+1] scratch offsets for tild_index_map / stage calls
    uint32_t* cell_fill;   // [max_bins+1] histogram
    uint32_t* scan_part;   // block sums for the scan, then rank[n]
    float* stage_x;        // [n][3] sorted copy of caller positions (stage calls)
    int32_t* stage_type;   // [n]
    float* tables;      // k-space tables

    cufftHandle plan_r2c, plan_c2r;
    bool plans_ok;

    bool has_state;
    uint64_t step;
    int steps_since_sort;
    int resort_every;
    int64_t launches;

    // timing
    cudaEvent_t ev[TILD_MAX_TIMED_STEPS][TILD_N_STAGE_EVENTS];
    bool ev_ok;
    int timed_steps;

    char err[512];
};

int tild_fail(tild_ctx* c, int code, const char* fmt, ...);
#define TILD_CUDA(c, call)                                                                          \
    do {                                                                                            \
        cudaError_t e__ = (call);                                                                   \
        if (e__ != cudaSuccess) return tild_fail((c), TILD_ECUDA, "%s: %s", #call, cudaGetErrorString(e__)); \
    } while (0)
#define TILD_LAUNCH_CHECK(c, name)                                                                  \
    do {                                                                                            \
        (c)->launches++;                                                                            \
        cudaError_t e__ = cudaGetLastError();                                                       \
        if (e__ != cudaSuccess) return tild_fail((c), TILD_ECUDA, "launch %s: %s", name, cudaGetErrorString(e__)); \
    } while (0)

// ---- stage launchers (each enqueues on c->stream) -----------------------------------------------
int launch_cell_keys(tild_ctx* c, const float* x, uint32_t* key, int32_t* base /*nullable*/);  // row-major cell keys
int launch_tile_keys(tild_ctx* c, const float* x, const int32_t* type, uint32_t* key);        // (tile, species, cell) keys
int launch_counting_sort(tild_ctx* c, const uint32_t* key, size_t nbins, uint32_t* perm, uint32_t* start);
int launch_reorder(tild_ctx* c);  // sorts the internal state by tile-major cell and flips buffers
int launch_stage_sort(tild_ctx* c, const float* x, const int32_t* type);  // caller arrays -> stage_x/stage_type + cell_start
int launch_spread_naive(tild_ctx* c, const float* x, const int32_t* type, float* grid);
int launch_spread_tiled(tild_ctx* c, const uint32_t* cell_start, const float* x, float* grid);
int tild_spread_configure(tild_ctx* c);
int launch_kspace(tild_ctx* c, const float2* nhat, float2* fhat);
int launch_interp_force(tild_ctx* c, const float* ffield, const float* x, const int32_t* type, float* f);
int launch_bond_force(tild_ctx* c, const float* x, const int32_t* bond, float* f, bool accumulate);
int launch_fused_step(tild_ctx* c);  // interp + bonds + GJF on the internal state, flips x/w buffers
int launch_make_w(tild_ctx* c, const float* f, float* w, float sign);  // w += sign*(dt/2m) f
int launch_philox_test(tild_ctx* c, const uint32_t* ctr, const uint32_t* key, uint32_t* out, float* gauss, int m);
int launch_unpermute(tild_ctx* c, const float* src, float* dst, int ncomp);  // dst[id[i]] = src[i]

size_t tild_scan_scratch_entries(size_t nbins, int n);

// ---- device helpers ------------------------------------------------------------------------------
#ifdef __CUDACC__

// Canonical fp32 index map of one coordinate (A15): every operation is a single correctly
// rounded fp32 operation (no FMA contraction).  Returns the cell (unwrapped floor), the first stencil
// node b (unwrapped) and the offset t in [-1/2, 1/2] from the stencil centre.
template <int P>
__device__ __forceinline__ void index_1d(float x, float inv_h, int& cell, int& b, float& t)
{
    const float s = __fmul_rn(x, inv_h);
    const float fl = floorf(s);
    cell = (int)fl;
    if (P % 2 == 0) {
        t = __fsub_rn(__fsub_rn(s, fl), 0.5f);
        b = cell - P / 2 + 1;
    } else {
        const float cp = floorf(__fadd_rn(s, 0.5f));
        t = __fsub_rn(s, cp);
        b = (int)cp - (P - 1) / 2;
    }
}

__device__ __forceinline__ int wrap_idx(int a, int N)
{
    a %= N;
    return a < 0 ? a + N : a;
}

// Order-P assignment weights (P-fold top-hat convolution; PAPER.md L223 -> Deserno & Holm appendix).
template <int P>
__device__ __forceinline__ void weights_1d(float t, float* w)
{
    if (P == 1) {
        w[0] = 1.0f;
    } else if (P == 2) {
        w[0] = 0.5f - t;
        w[1] = 0.5f + t;
    } else if (P == 3) {
        const float a = 0.5f - t, b = 0.5f + t;
        w[0] = 0.5f * a * a;
        w[1] = 0.75f - t * t;
        w[2] = 0.5f * b * b;
    } else {
        const float a = 1.0f - 2.0f * t, b = 1.0f + 2.0f * t;
        const float t2 = t * t;
        w[0] = a * a * a * (1.0f / 48.0f);
        w[3] = b * b * b * (1.0f / 48.0f);
        const float even = 23.0f - 12.0f * t2, odd = t * (24.0f * t2 - 30.0f);
        w[1] = (even + odd) * (1.0f / 48.0f);
        w[2] = (even - odd) * (1.0f / 48.0f);
    }
}

// Philox4x32-10 (Salmon et al., SC'11), written from the published round function.
__device__ __forceinline__ uint4 philox4x32_10(uint4 c, uint32_t k0, uint32_t k1)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c.x), lo0 = 0xD2511F53u * c.x;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c.z), lo1 = 0xCD9E8D57u * c.z;
        c = make_uint4(hi1 ^ c.y ^ k0, lo1, hi0 ^ c.w ^ k1, lo0);
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    return c;
}

// Three standard normals for (particle id, step): counter (id, step_lo, step_hi, 0); u = ((r>>9)+0.5) 2^-23
// (exact in fp32); Box-Muller (A12).
__device__ __forceinline__ float3 gauss3(uint32_t id, uint64_t step, uint32_t k0, uint32_t k1)
{
    const uint4 r = philox4x32_10(make_uint4(id, (uint32_t)step, (uint32_t)(step >> 32), 0u), k0, k1);
    const float sc = 1.0f / 8388608.0f;
    const float u0 = ((float)(r.x >> 9) + 0.5f) * sc, u1 = ((float)(r.y >> 9) + 0.5f) * sc;
    const float u2 = ((float)(r.z >> 9) + 0.5f) * sc, u3 = ((float)(r.w >> 9) + 0.5f) * sc;
    const float r01 = sqrtf(-2.0f * logf(u0)), r23 = sqrtf(-2.0f * logf(u2));
    float s1, c1;
    sincospif(2.0f * u1, &s1, &c1);
    return make_float3(r01 * c1, r01 * s1, r23 * cospif(2.0f * u3));
}

__device__ __forceinline__ float wrap_pos(float x, float L, float inv_L)
{
    float r = x - L * floorf(x * inv_L);
    if (r >= L) r -= L;
    if (r < 0.0f) r = 0.0f;
    if (r >= L) r = 0.0f;
    return r;
}

__device__ __forceinline__ float min_image(float d, float L, float inv_L)
{
    return d - L * rintf(d * inv_L);
}

#endif  // __CUDACC__
