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
    // layout of the force field the interpolation kernels read: node (x, y, z) of component c is at
    // ffield[c * FM + (x * FN[0] + y) * FN[1] + z].  Plain arrays: FN = (Ny, Nz), FM = M.  (A ghost-padded layout for TMA
    // staging was measured and dropped: cuFFT's C2R into padded rows costs more than the staging saves.)
    int FN[2];
    long long FM;
};

// Tiling of the cell grid.  A tile is T[0] x T[1] x T[2] cells; its shared-memory image holds
// E = T + H nodes per axis (H = stencil halo; in z also `sh` alignment nodes).  A "segment" is (tile, species):
// the internal particle arrays are kept sorted by segment, dense, in arbitrary order inside a segment.  Every step
// each tile kernel bins its own particles in shared memory by the BANK of the first stencil node's shared-memory
// address ("class", 32 of them) and then works in rounds of one particle per class, so that all 32 lanes of every
// stencil access hit different banks.
struct TileParams {
    int T[3];       // tile edge in cells (clipped to the grid)
    int nt[3];      // tiles per axis = ceil(N/T)
    int E[3];       // shared image edge in nodes: E[0] = T[0] + H, E[1] = T[1] + H (<= template EY), E[2] = EZ
    int lo;         // nodes below the tile's first cell that a stencil can touch (0 for P <= 2, 1 for P = 3, 4, 2 for P = 5)
    int sh;         // extra nodes below those so that the image starts on a 16-byte boundary of the mesh rows
    int H;          // stencil halo in nodes (1 for P <= 2, 3 for P = 3, 4, 5 for P = 5)
    int EY, EZ;     // template strides the kernels were instantiated with
    int ntiles;
    int nseg;       // ntiles * S
    int sp_group;   // species accumulated per spread CTA (shared-memory budget)
    size_t smem_spread, smem_interp;
    int enabled;    // 0: grid too small for the tile kernels -> per-particle kernels
};

// shared-memory particle binning of the tile kernels
#define TILD_SPREAD_CHUNK 4096   // particles binned at a time by the spread kernel (all species of its group)
#define TILD_SPREAD_KCAP 144     // rounds of its class lists (1.125 x the mean of a full chunk); the rest overflows
#define TILD_INTERP_CHUNK 2048   // same for the interpolation kernel (one species at a time)
#define TILD_INTERP_KCAP 96

struct KspaceParams {
    int S;
    int N[3];
    int Nzc;                 // Nz/2 + 1
    const float* kgrad[3];   // k_a(m), 0 at the Nyquist index of even N (A6)
    const float* ufac[3];    // exp(-sigma2 k_a(m)^2 / 2); ufac[0] also carries 1/V
    float c[TILD_MAX_SPECIES * TILD_MAX_SPECIES];  // c_IJ (1/V folded into ufac[0])
    // electrostatics (A22): u_el = eel[0] eel[1] eel[2] / (k2[0] + k2[1] + k2[2]), 0 at k = 0; 4 pi l_B / V in eel[0]
    int has_el;
    const float* eel[3];     // exp(-k_a^2 a_q^2) (times the deconvolution factor when that is on)
    const float* k2[3];      // k_a(m)^2, true wave number (Nyquist included)
    float qq[TILD_MAX_SPECIES * TILD_MAX_SPECIES];  // z_I z_J
    float sigma2, aq2;       // variance of u_G and a_q^2 (virial)
};

struct StepParams {
    float half_dt_over_m;  // dt/2m
    float kick_in;         // v^n = w^n + kick_in F^n: dt/2m, or 0 while the state still holds v itself (first step after tild_set_state)
    // One step of every inertial integrator is linear in (v, F, beta) (A24):
    //   r' = r + b_dt v + b_dt2_over_2m F + b_dt_over_2m beta,   w' = a_g (v + w_fr F) + b_over_m beta
    // GJF (A11):            b dt, b dt^2/2m, b dt/2m;  a, dt/2m, b/m        (a, b of Gronbech-Jensen & Farago)
    // VV + Langevin (A24):  c dt, dt^2/2m,   dt/2m;    c^2, dt/(2m c), (1 + c)/2m,   c = 1 - gamma dt/2m
    float a_g;
    float w_fr;
    float b_dt;
    float b_dt2_over_2m;
    float b_dt_over_2m;
    float b_over_m;
    int dim2;              // TILD_FLAG_2D: no force, noise or motion along z (A27)
    float noise_amp;       // sqrt(2 gamma kT dt); 0 disables the draw
    float k_bond, r0_bond;
    int max_bonds;
    uint32_t key0, key1;   // Philox key = seed lo, hi
    float lambda_wlc;      // cosine angle potential, Eq. 16 (0 = none; needs max_bonds == 2)
    float k_theta, theta0; // harmonic angle potential k_theta (theta - theta0)^2, Eq. 17 (0 = none; same triplets)
    int integrator;        // TILD_INTEGRATOR_*
    float em_drift;        // dt/gamma
    float em_noise;        // 1/gamma (times beta = noise_amp * z)
};

// ---- context -----------------------------------------------------------------------------------
// One segment-sorted ordering of a particle set: particles of segment g are slots [seg_base[g], seg_base[g+1]).
struct SegLayout {
    uint32_t* seg_base;  // device [nseg+1]
};

struct tild_ctx {
    tild_params prm;
    cudaStream_t stream;
    int device;           // the CUDA device that was current at tild_init: every entry point runs on it
    MeshParams mesh;
    KspaceParams ksp;
    StepParams stp;
    size_t M, Mk;
    TileParams tile;
    size_t max_bins;      // max(M, nseg*32): histogram length

    // carved from the caller's workspace.  Slot arrays have n entries.
    float4* X4[2];        // (x, y, z, type as int bits)
    float4* W4[2];        // (w_x, w_y, w_z, original id as uint bits)
    int32_t* B[2];        // [n][max_bonds] partner SLOTS, -1 = none
    int cur;
    float4* F4;           // [n] per-slot force scratch
    float4* SX4;          // [n] stage-call scratch: segment-sorted copy of caller particles; caller-order staging
    SegLayout lay, lay_stage;
    float* grid;          // [S][M]
    float2* nhat;         // [S][Mk]
    float2* fhat;         // [3S][Mk]
    float* ffield;        // [3S][M]
    uint32_t* key;        // [n] sort scratch
    uint32_t* rank;       // [n] sort scratch; between sorts: the drift list of launch_interp
    uint32_t* inv;        // [n] old slot -> new slot
    uint32_t* drift_count;  // [4]
    double* d_energy;       // [8] reduction targets of tild_energy / tild_virial
    uint64_t* d_step;       // device copy of `step` (read by the fused step kernels, advanced by a kernel)
    uint64_t h_step_upload; // staging for the asynchronous upload of d_step
    uint32_t* count;      // [max_bins+1] histogram
    uint32_t* start;      // [max_bins+1] scan output (cell_start of tild_index_map)
    uint32_t* scan_part;  // block sums of the scan
    uint32_t* perm;       // [n] tild_index_map scratch
    float* tables;        // k-space tables

    // extra mesh interactions (TILD_FLAG_EXTRAS; tild_extra.cu): per-particle charges and Maier-Saupe partners by particle id
    float* q_id;          // [n]
    int32_t* msp_id;      // [n] partner id of every LC centre, -1 = not a centre
    uint32_t* slot_of_id; // [n], refreshed at every re-sort
    float4* Fext;         // [n] per-slot extra force
    float4* xacc;         // [n] Phi u accumulator of the Maier-Saupe orientation force
    float* xr;            // [4][M] real meshes
    float2* xh;           // [5][Mk] spectra
    bool has_q, has_ms, x_active;   // x_active: the last launch_extra_forces filled Fext
    double rho0;
    cufftHandle plan_x_r2c, plan_x_c2r;   // 3-D, one field
    bool xplans_ok;

    cufftHandle plan_r2c, plan_c2r;   // 3-D, batched over species / force components (plan_c2r only when !xfft_R)
    cufftHandle plan_r2c_yz, plan_c2r_yz;   // 2-D over (y, z), batched over the x planes: used with the fused x-transform
    int xfft_R;           // threads per line (R2) of kspace_xfft_kernel (Nx = R1 R2), 0 = 3-D cuFFT plans + kspace_kernel
    const float2* xtw;    // exp(-2 pi i j / Nx), j < Nx
    bool plans_ok;

    alignas(64) unsigned char fmap[128];   // CUtensorMap of c->ffield with the image box of the rotation-class kernel
    bool tma_ok;

    bool has_state;
    bool step_advanced;   // the last launch_interp advanced the device step counter itself (tile path)
    cudaStream_t copy_stream = nullptr;   // tild_get_state: x goes to the host while F(x) is evaluated for v
    cudaEvent_t copy_ev[2] = {nullptr, nullptr};
    // tild_run_host_submit / _wait (TILD_FLAG_HOST_PIPELINE): device staging of the host batches and the streams of the copies
    float *hp_x = nullptr, *hp_v = nullptr;          // input staging [n][3] (one set: tild_set_state has consumed it when submit returns)
    int32_t *hp_t = nullptr, *hp_b = nullptr;        // [n], [n][max_bonds]
    float *hp_xo[2] = {nullptr, nullptr}, *hp_vo[2] = {nullptr, nullptr};   // output staging, one set per batch in flight
    cudaStream_t hp_in = nullptr, hp_out = nullptr;
    cudaEvent_t hp_ev_in = nullptr, hp_ev_done = nullptr, hp_ev_out[4] = {nullptr, nullptr, nullptr, nullptr};   // ev_out: one per batch, ring of 4
    uint64_t hp_submitted = 0, hp_waited = 0;
    bool lay_valid = false;         // c->lay describes the buffer X4[cur] (set by the first sort of a state): re-sorts keep the stayers' order
    bool grid_clean = false;        // c->grid is all zero: the drift kernel of the fused step cleared it for the next spread
    bool graph_leaves_clean = false;
    uint64_t step;
    int steps_since_sort;
    int resorts_since_defrag;   // re-sorts since the state was last sorted from particle-id order (launch_defrag)
    int resort_every;
    int64_t launches;

    // Graph replay: [0] the instantiated graph of two re-sort cycles, [1] of one cycle that starts with the return to
    // particle-id order (launch_defrag), each with the state it was captured in
    cudaGraphExec_t graph_exec[2];
    bool graph_ok[2];
    int graph_cur[2];
    float4* graph_x0[2];
    int64_t graph_launches[2];
    bool graph_leaves_clean2[2];

    // timing
    cudaEvent_t ev[TILD_MAX_TIMED_STEPS][TILD_N_STAGE_EVENTS];
    bool ev_ok;
    int timed_steps;          // steps whose events are recorded and not yet folded
    double ms_sum[8];         // folded stage times (sums over ms_steps steps): any number of steps can be timed
    long long ms_steps;

    char err[512];
};

int tild_fail(tild_ctx* c, int code, const char* fmt, ...);
cudaError_t tild_raise_smem_limit(const void* func, size_t bytes);   // tild_api.cu
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
// tild_sort.cu
int launch_cell_keys(tild_ctx* c, const float* x, uint32_t* key, int32_t* base /*nullable*/);  // row-major cell keys
int launch_counting_sort(tild_ctx* c, const uint32_t* key, size_t nbins, uint32_t* perm, uint32_t* start);
int launch_pack(tild_ctx* c, const float* x, const float* v, const int32_t* type, const int32_t* bond, float4* X4,
                float4* W4, int32_t* B);                                  // caller arrays -> slots [0, n), slot i = id i
// src slots [0, n) -> segment-sorted dst; fills lay->seg_base and c->inv (old slot -> new slot)
int launch_segment_sort(tild_ctx* c, const float4* X4src, float4* X4dst, SegLayout* lay);
int launch_reorder(tild_ctx* c);  // re-sorts the internal state by segment and flips buffers
int launch_defrag(tild_ctx* c);   // back to particle-id order + first sort (every TILD_DEFRAG_EVERY re-sorts)
#define TILD_DEFRAG_EVERY 5
#define TILD_DEFRAG_MIN_N (1 << 20)   // smaller states live in L2 whatever their order, and their steps are launch-bound
int launch_unpermute(tild_ctx* c, const float4* src, float* dst);
int launch_slot_ids(tild_ctx* c, uint32_t* id);                          // id[s] = original id of slot s        // dst[id[s]][0..2] = src[s].xyz
// tild_spread.cu
int tild_spread_configure(tild_ctx* c);
int launch_spread(tild_ctx* c, const SegLayout& lay, const float4* X4, float* grid);  // zero fill + tile kernel
// tild_kspace.cu
int launch_kspace(tild_ctx* c, const float2* nhat, float2* fhat);
int kspace_xfft_radix(int Nx, int S);
int tild_kspace_configure(tild_ctx* c);
int launch_kspace_xfft(tild_ctx* c, const float2* nhat, float2* fhat);
// tild_interp.cu
int tild_interp_configure(tild_ctx* c);
enum { INTERP_NONBONDED_BY_ID = 0, INTERP_TOTAL_BY_SLOT = 1, INTERP_FUSED_STEP = 2 };
// mode 0: fout[id][3] = interpolated force; mode 1: c->F4[slot] = interpolated + bond force; mode 2: GJF step
int launch_interp(tild_ctx* c, int mode, const SegLayout& lay, const float* ffield, const float4* X4, const float4* W4,
                  const int32_t* B, float4* X4o, float4* W4o, float* fout);
int launch_bond_force_caller(tild_ctx* c, const float* x, const int32_t* bond, float* f);  // caller-order stage call
int launch_make_w(tild_ctx* c, const float4* F4, float4* W4, float sign);   // w += sign*(dt/2m) f
int launch_velocity_out(tild_ctx* c, const float4* F4, const float4* W4, float* v);  // v[id] = w + (dt/2m) f
int launch_advance_step(tild_ctx* c);
int launch_energy(tild_ctx* c, double* d_out);   // tild_energy.cu
// tild_extra.cu
int launch_slot_of_id(tild_ctx* c);
int launch_extra_forces(tild_ctx* c, const float4* X4, const float4* W4);
// adds the effect of Fext to what launch_interp produced: mode 1 the per-slot force F4, mode 2 the new state (X4o, W4o)
int launch_extra_apply(tild_ctx* c, int mode, float kick_in, float4* X4o, float4* W4o);
int launch_structure_factor(tild_ctx* c, uint32_t mask, float* sk, int accumulate);  // c->nhat must be current
int launch_philox_test(tild_ctx* c, const uint32_t* ctr, const uint32_t* key, uint32_t* out, float* gauss, int m);

struct InterpArgs {
    MeshParams m;
    TileParams tp;
    StepParams s;
    const uint64_t* step_ptr;
    const uint32_t* seg_base;
    const float* ffield;
    const float4* X4;
    const float4* W4;
    const int32_t* B;
    float4* X4o;
    float4* W4o;
    float4* F4;
    uint32_t* drift_list;
    uint32_t* drift_count;   // [0] entries of drift_list, [1] blocks of the drift kernel that are done
    uint64_t* step_adv;      // device step counter, advanced by the last block of the drift kernel in the fused step
    const void* fmap;        // CUtensorMap of the force field (tild_interp_rot.cu) when use_tma
    int use_tma;
    float4* zgrid;           // fused step: the density grid, cleared by the drift kernel for the next step's spread (or null)
    size_t zcount4;
};
// tild_spread_rot.cu: the P = 4 rotation-class spread kernel
bool spread_rot_applies(const tild_ctx* c);
cudaError_t spread_rot_run(const tild_ctx* c, const uint32_t* seg_base, const float4* X4, float* grid, bool configure_only);
// tild_interp_rot.cu: the P = 4 rotation-class tile kernel
bool interp_rot_applies(const tild_ctx* c);
bool interp_rot_make_tmap(tild_ctx* c);
size_t interp_rot_smem(int ey, int ez);
cudaError_t interp_rot_run(const InterpArgs& a, int mode, cudaStream_t st, bool configure_only);

size_t tild_scan_scratch_entries(size_t nbins);

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

// a in [-N, 2N): one conditional wrap each way (no integer division)
__device__ __forceinline__ int wrap_near(int a, int N)
{
    a += a < 0 ? N : 0;
    a -= a >= N ? N : 0;
    return a;
}

// any a; the integer division only runs for indices more than one period away (images wider than a tiny mesh)
__device__ __forceinline__ int wrap_idx(int a, int N)
{
    if ((unsigned)(a + N) < 3u * (unsigned)N) return wrap_near(a, N);
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
    } else if (P == 4) {
        const float a = 1.0f - 2.0f * t, b = 1.0f + 2.0f * t;
        const float t2 = t * t;
        w[0] = a * a * a * (1.0f / 48.0f);
        w[3] = b * b * b * (1.0f / 48.0f);
        const float even = 23.0f - 12.0f * t2, odd = t * (24.0f * t2 - 30.0f);
        w[1] = (even + odd) * (1.0f / 48.0f);
        w[2] = (even - odd) * (1.0f / 48.0f);
    } else {   // P = 5 (the paper's "order 4", A1): quartic B-spline
        const float a = 1.0f - 2.0f * t, b = 1.0f + 2.0f * t;
        const float t2 = t * t, a2 = a * a, b2 = b * b;
        w[0] = a2 * a2 * (1.0f / 384.0f);
        w[4] = b2 * b2 * (1.0f / 384.0f);
        const float even = 19.0f + t2 * (24.0f - 16.0f * t2), odd = t * (16.0f * t2 - 44.0f);
        w[1] = (even + odd) * (1.0f / 96.0f);
        w[3] = (even - odd) * (1.0f / 96.0f);
        w[2] = (115.0f + t2 * (48.0f * t2 - 120.0f)) * (1.0f / 192.0f);
    }
}

// stencil halo of order P relative to the particle's cell: nodes [cell - LO, cell - LO + H + 1)
template <int P> struct Halo {
    static constexpr int H = P <= 2 ? 1 : (P <= 4 ? 3 : 5);     // extra nodes a tile image needs per axis
    static constexpr int LO = P <= 2 ? 0 : (P <= 4 ? 1 : 2);    // of which below the tile's first cell
    static constexpr int EZA = P <= 2 ? 20 : 24, EZB = P <= 2 ? 36 : 40;   // image z extent for TZ = 16 / 32 (% 4 == 0)
};

// Packed fp32 pair arithmetic (sm_100a: FFMA2 / FMUL2, one issue slot for two lanes of a register pair).
// d = a * b + c with b broadcast to both halves: ptxas folds the duplicate into the scalar-broadcast operand form.
__device__ __forceinline__ float2 ffma2_bcast(float2 a, float b, float2 c)
{
#ifndef TILD_USE_FFMA2
    return make_float2(fmaf(a.x, b, c.x), fmaf(a.y, b, c.y));
#endif
    unsigned long long ra, rb, rc, rd;
    asm("mov.b64 %0, {%1, %2};" : "=l"(ra) : "f"(a.x), "f"(a.y));
    asm("mov.b64 %0, {%1, %1};" : "=l"(rb) : "f"(b));
    asm("mov.b64 %0, {%1, %2};" : "=l"(rc) : "f"(c.x), "f"(c.y));
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(rd) : "l"(ra), "l"(rb), "l"(rc));
    float2 d;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(d.x), "=f"(d.y) : "l"(rd));
    return d;
}
__device__ __forceinline__ float2 fmul2_bcast(float2 a, float b)
{
    unsigned long long ra, rb, rd;
    asm("mov.b64 %0, {%1, %2};" : "=l"(ra) : "f"(a.x), "f"(a.y));
    asm("mov.b64 %0, {%1, %1};" : "=l"(rb) : "f"(b));
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(rd) : "l"(ra), "l"(rb));
    float2 d;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(d.x), "=f"(d.y) : "l"(rd));
    return d;
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
// (exact in fp32); Box-Muller (A12).  The transcendental functions are the hardware approximations
// (MUFU.LG2 / SQRT / SIN / COS: absolute error <= 2^-20.9 on the unit circle, 2^-22 in lg2), which keeps the draw at
// ~10 instead of ~130 instructions; the deviation from the correctly rounded value is < 3e-6 per normal, i.e. < 1e-9
// in a position per step.  Angles are taken in [-pi, pi) where the approximation is specified.
__device__ __forceinline__ float sqrt_approx(float x)
{
    float r;
    asm("sqrt.approx.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ float3 gauss3(uint32_t id, uint64_t step, uint32_t k0, uint32_t k1)
{
    const uint4 r = philox4x32_10(make_uint4(id, (uint32_t)step, (uint32_t)(step >> 32), 0u), k0, k1);
    const float sc = 1.0f / 8388608.0f, hs = 0.5f / 8388608.0f;
    const float u0 = fmaf((float)(r.x >> 9), sc, hs), u2 = fmaf((float)(r.z >> 9), sc, hs);
    // 2 pi (u - 1/2): (r >> 9) 2^-23 - 1/2 + 2^-24 is exact in fp32
    const float a1 = 6.283185307179586f * (fmaf((float)(r.y >> 9), sc, hs) - 0.5f);
    const float a3 = 6.283185307179586f * (fmaf((float)(r.w >> 9), sc, hs) - 0.5f);
    const float r01 = sqrt_approx(-1.3862943611198906f * __log2f(u0));   // sqrt(-2 ln u) = sqrt(-2 ln2 lg2 u)
    const float r23 = sqrt_approx(-1.3862943611198906f * __log2f(u2));
    // cos(2 pi u) = -cos(2 pi (u - 1/2)), likewise sin
    return make_float3(-r01 * __cosf(a1), -r01 * __sinf(a1), -r23 * __cosf(a3));
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

// Gradients of cos(theta) = d1.d2 / (|d1| |d2|) with respect to the end points of d1 and d2 (Eq. 16):
// gi = d cos / d r_i = d2 / (|d1||d2|) - cos d1 / |d1|^2,  gk likewise;  d cos / d r_j = -(gi + gk).  Returns cos.
__device__ __forceinline__ float cos_gradients(const float d1[3], const float d2[3], float gi[3], float gk[3], float& sn)
{
    sn = 0.0f;
    const float n1 = d1[0] * d1[0] + d1[1] * d1[1] + d1[2] * d1[2], n2 = d2[0] * d2[0] + d2[1] * d2[1] + d2[2] * d2[2];
    if (!(n1 > 0.0f) || !(n2 > 0.0f)) {
        gi[0] = gi[1] = gi[2] = gk[0] = gk[1] = gk[2] = 0.0f;
        return -1.0f;
    }
    const float inv = rsqrtf(n1) * rsqrtf(n2), c = (d1[0] * d2[0] + d1[1] * d2[1] + d1[2] * d2[2]) * inv;
    const float c1 = c / n1, c2 = c / n2;
    const float cx = d1[1] * d2[2] - d1[2] * d2[1], cy = d1[2] * d2[0] - d1[0] * d2[2], cz = d1[0] * d2[1] - d1[1] * d2[0];
    sn = sqrtf(cx * cx + cy * cy + cz * cz) * inv;    // sin(theta) from the cross product: no cancellation near 0 and pi
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        gi[a] = d2[a] * inv - c1 * d1[a];
        gk[a] = d1[a] * inv - c2 * d2[a];
    }
    return c;
}

// dU/d(cos theta) of U = lambda (1 + cos theta) + k_theta (theta - theta0)^2 (Eq. 16-17):
// lambda - 2 k_theta (theta - theta0) / sin theta, theta = atan2(sin, cos).  The harmonic term is singular at
// sin theta -> 0 (unless theta0 is that angle) and is dropped there.
__device__ __forceinline__ float angle_dUdc(float lambda, float k_theta, float theta0, float c, float sn)
{
    float coef = lambda;
    if (k_theta != 0.0f && sn > 1e-6f) coef -= 2.0f * k_theta * (atan2f(sn, c) - theta0) / sn;
    return coef;
}

// Force of the angle potentials on the bead at r with neighbours: prev / next (either may be missing) and their
// own outer neighbours pprev / nnext.  has_* say which exist.  Each bead computes its own share of the (up to) three
// angles it belongs to, without Newton's third law (as the paper does for bonds, L209).
__device__ __forceinline__ void wlc_angle_force(float lambda, float k_theta, float theta0, const float L[3], const float inv_L[3], const float r[3],
                                                bool has_prev, const float prev[3], bool has_pprev, const float pprev[3],
                                                bool has_next, const float next[3], bool has_nnext, const float nnext[3],
                                                float f[3])
{
    float d1[3], d2[3], gi[3], gk[3], sn, c, coef;
    if (has_prev && has_next) {          // centre bead of (prev, r, next)
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            d1[a] = min_image(prev[a] - r[a], L[a], inv_L[a]);
            d2[a] = min_image(next[a] - r[a], L[a], inv_L[a]);
        }
        c = cos_gradients(d1, d2, gi, gk, sn);
        coef = angle_dUdc(lambda, k_theta, theta0, c, sn);
#pragma unroll
        for (int a = 0; a < 3; ++a) f[a] += coef * (gi[a] + gk[a]);
    }
    if (has_prev && has_pprev) {         // end bead k of (pprev, prev, r)
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            d1[a] = min_image(pprev[a] - prev[a], L[a], inv_L[a]);
            d2[a] = min_image(r[a] - prev[a], L[a], inv_L[a]);
        }
        c = cos_gradients(d1, d2, gi, gk, sn);
        coef = angle_dUdc(lambda, k_theta, theta0, c, sn);
#pragma unroll
        for (int a = 0; a < 3; ++a) f[a] -= coef * gk[a];
    }
    if (has_next && has_nnext) {         // end bead i of (r, next, nnext)
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            d1[a] = min_image(r[a] - next[a], L[a], inv_L[a]);
            d2[a] = min_image(nnext[a] - next[a], L[a], inv_L[a]);
        }
        c = cos_gradients(d1, d2, gi, gk, sn);
        coef = angle_dUdc(lambda, k_theta, theta0, c, sn);
#pragma unroll
        for (int a = 0; a < 3; ++a) f[a] -= coef * gi[a];
    }
}

#endif  // __CUDACC__
