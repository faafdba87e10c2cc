// C-ABI of libtild (include/tild.h): context, workspace carving, cuFFT plans, stage calls and the timed step.
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <map>
#include <mutex>
#include <new>
#include <utility>
#include <vector>

#include "tild_internal.cuh"

int tild_fail(tild_ctx* c, int code, const char* fmt, ...)
{
    if (c) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(c->err, sizeof(c->err), fmt, ap);
        va_end(ap);
    }
    return code;
}

// cudaFuncAttributeMaxDynamicSharedMemorySize is per FUNCTION and process-wide: contexts with different needs for the same
// kernel instantiation must never lower it (a later tild_init would otherwise break an earlier context's launches).
// Raises the limit of `func` to at least `bytes`; keeps the maximum asked for so far per (device, function).
cudaError_t tild_raise_smem_limit(const void* func, size_t bytes)
{
    static std::mutex mu;
    static std::map<std::pair<int, const void*>, size_t> limit;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    std::lock_guard<std::mutex> lock(mu);
    size_t& cur = limit[std::make_pair(dev, func)];
    if (bytes <= cur) return cudaSuccess;
    e = cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    if (e == cudaSuccess) cur = bytes;
    return e;
}

namespace {

// Every entry point runs on the device that was current at tild_init, whatever is current on the calling thread.
struct DevGuard {
    int prev = 0;
    bool switched = false;
    explicit DevGuard(const tild_ctx* c)
    {
        if (c && cudaGetDevice(&prev) == cudaSuccess && prev != c->device) switched = cudaSetDevice(c->device) == cudaSuccess;
    }
    ~DevGuard()
    {
        if (switched) cudaSetDevice(prev);
    }
};

constexpr size_t ALIGN = 256;
inline size_t up(size_t b) { return (b + ALIGN - 1) / ALIGN * ALIGN; }

// Walks the workspace layout; with base == nullptr it only measures.
struct Carver {
    char* base;
    size_t off = 0;
    explicit Carver(void* b) : base(static_cast<char*>(b)) {}
    template <typename T>
    T* take(size_t count)
    {
        T* p = base ? reinterpret_cast<T*>(base + off) : nullptr;
        off += up(count * sizeof(T) + 16);
        return p;
    }
};

int validate(const tild_params* p)
{
    if (!p || p->struct_size != sizeof(tild_params)) return TILD_EINVAL;
    if (p->n < 0 || p->n_species < 1 || p->n_species > TILD_MAX_SPECIES) return TILD_EINVAL;
    if (p->order < 1 || p->order > 5) return TILD_EINVAL;
    if (p->max_bonds < 0 || p->max_bonds > TILD_MAX_BONDS) return TILD_EINVAL;
    double M = 1.0;
    for (int a = 0; a < 3; ++a) {
        const bool flat = a == 2 && (p->flags & TILD_FLAG_2D);          // 2-D mode: one plane of nodes, any order
        if (flat && p->grid[a] != 1) return TILD_EINVAL;
        if (!(p->box[a] > 0.0) || (!flat && (p->grid[a] < p->order || p->grid[a] < 2)) || p->grid[a] > 4096) return TILD_EINVAL;
        M *= p->grid[a];
    }
    if (M > 2.0e9) return TILD_EINVAL;
    if (!(p->sigma2 > 0.0) && !(p->a > 0.0)) return TILD_EINVAL;
    if (!(p->dt > 0.0) || !(p->mass > 0.0) || p->gamma < 0.0 || p->kT < 0.0) return TILD_EINVAL;
    if (p->integrator != TILD_INTEGRATOR_GJF && p->integrator != TILD_INTEGRATOR_EM && p->integrator != TILD_INTEGRATOR_VV) return TILD_EINVAL;
    if (p->integrator == TILD_INTEGRATOR_VV && !(p->gamma * p->dt / (2.0 * p->mass) < 1.0)) return TILD_EINVAL;   // c = 1 - gamma dt/2m > 0
    if (p->integrator == TILD_INTEGRATOR_EM && !(p->gamma > 0.0)) return TILD_EINVAL;
    if ((p->lambda_wlc != 0.0 || p->k_theta != 0.0) && p->max_bonds != 2) return TILD_EINVAL;
    if (!(p->k_theta >= 0.0) || !(p->theta0 >= 0.0 && p->theta0 <= 3.141592653589794)) return TILD_EINVAL;
    if (p->bjerrum < 0.0 || (p->bjerrum > 0.0 && !(p->a_charge > 0.0))) return TILD_EINVAL;
    return TILD_OK;
}

// Tile shape: 8 x TY x TZ cells, TY in {8, 16} (template EY = TY + H), TZ in {16, 32}; the shared
// image is EZ = TZ + H + sh nodes long in z, rounded up to a multiple of 4.  tild_params.tile_shape = TY | TZ << 8
// selects another shape than the default 8 x 16 x 32 (0 = default).
void configure_tiles(tild_ctx* c)
{
    const tild_params& p = c->prm;
    TileParams& t = c->tile;
    memset(&t, 0, sizeof(t));
    t.H = p.order <= 2 ? 1 : (p.order <= 4 ? 3 : 5);
    t.lo = p.order <= 2 ? 0 : (p.order <= 4 ? 1 : 2);
    t.sh = t.lo ? 4 - t.lo : 0;   // image starts on a 16-byte boundary of the mesh rows (16-byte cp.async staging)
    t.enabled = p.grid[0] >= 8 && p.grid[1] >= 8 && p.grid[2] >= 8;
    const int tx = 8;
    int ty = p.tile_shape & 0xff, tz = (p.tile_shape >> 8) & 0xff;
    const bool auto_y = ty != 8 && ty != 16, auto_z = tz != 16 && tz != 32;
    if (auto_y) ty = 16;
    if (auto_z) tz = p.grid[2] >= 32 ? 32 : 16;
    // Default shape 8 x 16 x 32, halved in y and then in z while the tiles are too few to fill the GPU (two CTAs per SM on
    // 148 SMs) or hold more than 4096 particles each (several chunks per species and image, and few, long CTAs: measured on
    // the C5 sweep at 128^3, 8192 particles per tile: step 0.600 -> 0.475 ms at P = 4, 0.540 -> 0.397 ms at P = 3; C2 at 64^3,
    // 64 tiles: 0.082 -> 0.075 ms; C3 and C4 with 2048 particles in each of 512 / 4096 tiles keep the default)
    if (auto_y || auto_z) {
        auto crowded = [&](int y, int z) {
            const long long nt = (long long)((p.grid[0] + tx - 1) / tx) * ((p.grid[1] + y - 1) / y) * ((p.grid[2] + z - 1) / z);
            return nt < 296 || (long long)p.n > 4096 * nt;
        };
        if (auto_y && crowded(ty, tz)) ty = 8;
        if (auto_z && tz == 32 && crowded(ty, tz)) tz = 16;
    }
    const int ez = (tz + t.H + t.sh + 3) / 4 * 4;
    const size_t lists_i = (size_t)TILD_INTERP_KCAP * 32 * 2 + (size_t)TILD_INTERP_CHUNK * 2;
    const size_t lists_s = (size_t)TILD_SPREAD_KCAP * 32 * 4 + (size_t)TILD_SPREAD_CHUNK * 4;
    t.EY = ty + t.H;
    t.EZ = ez;
    const int T[3] = {tx, ty, tz};
    t.ntiles = 1;
    for (int a = 0; a < 3; ++a) {
        t.T[a] = T[a] < p.grid[a] ? T[a] : p.grid[a];
        t.nt[a] = (p.grid[a] + t.T[a] - 1) / t.T[a];
        t.E[a] = t.T[a] + t.H;
        t.ntiles *= t.nt[a];
    }
    t.E[2] = ez;
    t.nseg = t.ntiles * p.n_species;
    const size_t per_species = (size_t)t.E[0] * t.EY * t.EZ * sizeof(uint32_t);
    t.sp_group = (int)((100 * 1024 - lists_s) / per_species);
    if (t.sp_group < 1) t.sp_group = 1;
    if (t.sp_group > p.n_species) t.sp_group = p.n_species;
    t.smem_spread = per_species * t.sp_group + lists_s;
    t.smem_interp = (size_t)t.E[0] * t.EY * 3 * t.EZ * sizeof(float) + lists_i;
    const size_t M = (size_t)p.grid[0] * p.grid[1] * p.grid[2];
    c->max_bins = M > (size_t)t.nseg ? M : (size_t)t.nseg;
    if (c->max_bins < 2 * (size_t)t.nseg + 4) c->max_bins = 2 * (size_t)t.nseg + 4;   // re-sort: two arrays per segment in count / start
}

void carve(tild_ctx* c, void* base, size_t* total)
{
    configure_tiles(c);
    const tild_params& p = c->prm;
    const size_t n = (size_t)p.n, S = (size_t)p.n_species;
    const size_t M = (size_t)p.grid[0] * p.grid[1] * p.grid[2];
    const size_t Mk = (size_t)p.grid[0] * p.grid[1] * (p.grid[2] / 2 + 1);
    const size_t nb = n * (size_t)(p.max_bonds > 0 ? p.max_bonds : 1);
    Carver w(base);
    for (int k = 0; k < 2; ++k) {
        c->X4[k] = w.take<float4>(n);
        c->W4[k] = w.take<float4>(n);
        c->B[k] = w.take<int32_t>(nb);
    }
    c->F4 = w.take<float4>(n);
    c->SX4 = w.take<float4>(n);
    c->lay.seg_base = w.take<uint32_t>((size_t)c->tile.nseg + 2);
    c->lay_stage.seg_base = w.take<uint32_t>((size_t)c->tile.nseg + 2);
    c->grid = w.take<float>(S * M);
    c->nhat = w.take<float2>(S * Mk);
    c->fhat = w.take<float2>(3 * S * Mk);
    c->ffield = w.take<float>(3 * S * M);
    c->key = w.take<uint32_t>(n);
    c->rank = w.take<uint32_t>(n);
    c->inv = w.take<uint32_t>(n);
    c->count = w.take<uint32_t>(c->max_bins + 2);
    c->start = w.take<uint32_t>(c->max_bins + 2);
    c->scan_part = w.take<uint32_t>(tild_scan_scratch_entries(c->max_bins + 2));
    c->perm = w.take<uint32_t>(n);
    c->drift_count = w.take<uint32_t>(4);
    c->d_step = w.take<uint64_t>(2);
    c->d_energy = w.take<double>(8);
    c->tables = w.take<float>(14 * 4096);
    if (p.flags & TILD_FLAG_HOST_PIPELINE) {   // tild_run_host_submit: staging of the host batches
        c->hp_x = w.take<float>(3 * n);
        c->hp_v = w.take<float>(3 * n);
        c->hp_t = w.take<int32_t>(n);
        c->hp_b = w.take<int32_t>(nb);
        for (int k = 0; k < 2; ++k) {
            c->hp_xo[k] = w.take<float>(3 * n);
            c->hp_vo[k] = w.take<float>(3 * n);
        }
    }
    if (p.flags & TILD_FLAG_EXTRAS) {   // per-particle charges / Maier-Saupe (tild_extra.cu)
        c->q_id = w.take<float>(n);
        c->msp_id = w.take<int32_t>(n);
        c->slot_of_id = w.take<uint32_t>(n);
        c->Fext = w.take<float4>(n);
        c->xacc = w.take<float4>(n);
        c->xr = w.take<float>(4 * M);
        c->xh = w.take<float2>(5 * Mk);
    }
    *total = w.off;
}

#define TILD_FFT(c, call)                                                                  \
    do {                                                                                   \
        cufftResult r__ = (call);                                                          \
        if (r__ != CUFFT_SUCCESS) return tild_fail((c), TILD_ECUFFT, "%s: cufft error %d", #call, (int)r__); \
    } while (0)

// out[i][0..2] = F4[inv[i]].xyz: per-slot results of a stage call back to caller order (inv: source slot = id -> slot)
__global__ void __launch_bounds__(256) gather_by_inv_kernel(int n, const uint32_t* __restrict__ inv, const float4* __restrict__ F4,
                                                            float* __restrict__ out)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float4 f = F4[inv[i]];
    out[3 * (size_t)i + 0] = f.x;
    out[3 * (size_t)i + 1] = f.y;
    out[3 * (size_t)i + 2] = f.z;
}

// R2C -> k-space multiplication -> C2R.  With the fused x-transform (xfft_R) cuFFT runs over (y, z) only and
// kspace_xfft_kernel does the x transforms around the multiplication; otherwise 3-D plans and kspace_kernel.
int kspace_pipeline(tild_ctx* c, const float* grid, float* ffield, cudaEvent_t* ev)
{
    int rc;
    cufftComplex* nh = reinterpret_cast<cufftComplex*>(c->nhat);
    cufftComplex* fh = reinterpret_cast<cufftComplex*>(c->fhat);
    if (c->xfft_R) {
        TILD_FFT(c, cufftExecR2C(c->plan_r2c_yz, const_cast<float*>(grid), nh));
        if (ev) TILD_CUDA(c, cudaEventRecord(ev[3], c->stream));
        rc = launch_kspace_xfft(c, c->nhat, c->fhat);
        if (rc) return rc;
        if (ev) TILD_CUDA(c, cudaEventRecord(ev[4], c->stream));
        TILD_FFT(c, cufftExecC2R(c->plan_c2r_yz, fh, ffield));
    } else {
        TILD_FFT(c, cufftExecR2C(c->plan_r2c, const_cast<float*>(grid), nh));
        if (ev) TILD_CUDA(c, cudaEventRecord(ev[3], c->stream));
        rc = launch_kspace(c, c->nhat, c->fhat);
        if (rc) return rc;
        if (ev) TILD_CUDA(c, cudaEventRecord(ev[4], c->stream));
        TILD_FFT(c, cufftExecC2R(c->plan_c2r, fh, ffield));
    }
    if (ev) TILD_CUDA(c, cudaEventRecord(ev[5], c->stream));
    return TILD_OK;
}

// spread -> R2C -> k-space -> C2R on slab-ordered particles, with optional stage events
int mesh_pipeline(tild_ctx* c, const SegLayout& lay, const float4* X4, cudaEvent_t* ev)
{
    int rc = launch_spread(c, lay, X4, c->grid);
    if (rc) return rc;
    if (ev) TILD_CUDA(c, cudaEventRecord(ev[2], c->stream));
    return kspace_pipeline(c, c->grid, c->ffield, ev);
}

// total force at the current internal positions -> c->F4 (per slot); no state change
int force_current(tild_ctx* c)
{
    const int a = c->cur;
    int rc = mesh_pipeline(c, c->lay, c->X4[a], nullptr);
    if (rc) return rc;
    if ((rc = launch_extra_forces(c, c->X4[a], c->W4[a]))) return rc;
    if ((rc = launch_interp(c, INTERP_TOTAL_BY_SLOT, c->lay, c->ffield, c->X4[a], c->W4[a], c->B[a], nullptr, nullptr, nullptr))) return rc;
    return launch_extra_apply(c, 1, 0.0f, nullptr, nullptr);
}

// caller (x, type) -> segment-sorted copy in c->SX4 described by c->lay_stage; c->inv maps id -> slot
int stage_layout(tild_ctx* c, const float* x, const int32_t* type)
{
    int rc = launch_pack(c, x, nullptr, type, nullptr, c->F4, nullptr, nullptr);
    if (rc) return rc;
    return launch_segment_sort(c, c->F4, c->SX4, &c->lay_stage);
}

// the instantiated graphs have the current choice of extra interactions baked in
void drop_graphs(tild_ctx* c)
{
    for (int g = 0; g < 2; ++g)
        if (c->graph_ok[g]) {
            cudaGraphExecDestroy(c->graph_exec[g]);
            c->graph_ok[g] = false;
        }
}

}  // namespace

extern "C" {

const char* tild_version(void) { return "tild-b200 0.1 (sm_100a)"; }

int tild_workspace_bytes(const tild_params* params, size_t* bytes)
{
    if (!bytes) return TILD_EINVAL;
    int rc = validate(params);
    if (rc) return rc;
    tild_ctx tmp;
    memset(&tmp, 0, sizeof(tmp));
    tmp.prm = *params;
    carve(&tmp, nullptr, bytes);
    return TILD_OK;
}

int tild_init(tild_ctx** out, const tild_params* params, void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    if (!out) return TILD_EINVAL;
    *out = nullptr;
    int rc = validate(params);
    if (rc) return rc;
    if (!workspace || (reinterpret_cast<uintptr_t>(workspace) % ALIGN) != 0) return TILD_ENOMEM;
    tild_ctx* c = new (std::nothrow) tild_ctx;
    if (!c) return TILD_ENOMEM;
    memset(c, 0, sizeof(*c));
    c->prm = *params;
    c->stream = static_cast<cudaStream_t>(cuda_stream);
    if (cudaGetDevice(&c->device) != cudaSuccess) {
        delete c;
        return TILD_ECUDA;
    }
    size_t need = 0;
    carve(c, workspace, &need);
    if (need > workspace_bytes) {
        delete c;
        return TILD_ENOMEM;
    }
    const tild_params& p = c->prm;
    const int S = p.n_species;
    c->M = (size_t)p.grid[0] * p.grid[1] * p.grid[2];
    c->Mk = (size_t)p.grid[0] * p.grid[1] * (p.grid[2] / 2 + 1);
    const double V = p.box[0] * p.box[1] * p.box[2];
    const double sigma2 = p.sigma2 > 0.0 ? p.sigma2 : 2.0 * p.a * p.a;
    const double rho0 = p.rho0 > 0.0 ? p.rho0 : (p.n > 0 ? (double)p.n / V : 1.0);   // L121; an empty system has no density scale
    c->resort_every = p.resort_every > 0 ? p.resort_every : 10;
    c->rho0 = rho0;

    MeshParams& m = c->mesh;
    m.n = p.n;
    m.S = S;
    m.P = p.order;
    m.M = (long long)c->M;
    m.FN[0] = p.grid[1];
    m.FN[1] = p.grid[2];
    m.FM = (long long)c->M;
    for (int a = 0; a < 3; ++a) {
        m.N[a] = p.grid[a];
        m.inv_h[a] = (float)((double)p.grid[a] / p.box[a]);
        m.L[a] = (float)p.box[a];
        m.inv_L[a] = (float)(1.0 / p.box[a]);
    }

    // a0: k-space tables in double on the host (A4-A6), uploaded as fp32
    std::vector<float> tab(14 * 4096, 0.0f);
    const double PI = 3.14159265358979323846264338327950288;
    for (int a = 0; a < 3; ++a) {
        const int N = p.grid[a];
        for (int mm = 0; mm < N; ++mm) {
            const int mt = mm <= N / 2 ? mm : mm - N;
            const double k = 2.0 * PI * (double)mt / p.box[a];
            const double kg = (N % 2 == 0 && mm == N / 2) ? 0.0 : k;
            double u = exp(-0.5 * sigma2 * k * k);
            if (p.flags & TILD_FLAG_SAMPLED_KERNEL) {
                // A5b: u_G sampled at the nodes with the minimum-image distance is a product of three 1-D Gaussians, so
                // its 3-D DFT is the product of three 1-D DFTs: u_a(m) = h sum_g g1(d_g) cos(2 pi m g / N)
                const double h = p.box[a] / (double)N;
                u = 0.0;
                for (int g = 0; g < N; ++g) {
                    double d = g * h;
                    if (d > 0.5 * p.box[a]) d -= p.box[a];
                    u += exp(-0.5 * d * d / sigma2) * cos(2.0 * PI * (double)mm * (double)g / (double)N);
                }
                u *= h / sqrt(2.0 * PI * sigma2);
            }
            if (p.flags & TILD_FLAG_DECONVOLVE) {   // separable: [sinc(k h / 2)]^(-2P) per axis
                const double xh = 0.5 * k * p.box[a] / (double)N;
                const double sinc = xh == 0.0 ? 1.0 : sin(xh) / xh;
                u /= pow(sinc, 2.0 * p.order);
            }
            if (a == 0) u /= V;
            tab[(size_t)a * 4096 + mm] = (float)kg;
            tab[(size_t)(3 + a) * 4096 + mm] = (float)u;
            // electrostatics (A22): separable Gaussian part of 4 pi l_B exp(-k^2 a_q^2) / k^2, and k_a^2
            double e = exp(-k * k * p.a_charge * p.a_charge);
            if (p.flags & TILD_FLAG_DECONVOLVE) {
                const double xh = 0.5 * k * p.box[a] / (double)N;
                const double sinc = xh == 0.0 ? 1.0 : sin(xh) / xh;
                e /= pow(sinc, 2.0 * p.order);
            }
            if (a == 0) e *= 4.0 * PI * p.bjerrum / V;
            tab[(size_t)(6 + a) * 4096 + mm] = (float)e;
            tab[(size_t)(9 + a) * 4096 + mm] = (float)(k * k);
        }
    }
    for (int j = 0; j < p.grid[0]; ++j) {      // x twiddles of the fused x-transform kernel
        const double ang = 2.0 * PI * (double)j / (double)p.grid[0];
        tab[(size_t)12 * 4096 + 2 * j] = (float)cos(ang);
        tab[(size_t)12 * 4096 + 2 * j + 1] = (float)(-sin(ang));
    }
    c->xtw = reinterpret_cast<const float2*>(c->tables + (size_t)12 * 4096);
    c->xfft_R = (p.flags & (TILD_FLAG_PLAIN_FFT | TILD_FLAG_2D)) ? 0 : kspace_xfft_radix(p.grid[0], S);
    KspaceParams& ks = c->ksp;
    ks.S = S;
    ks.Nzc = p.grid[2] / 2 + 1;
    for (int a = 0; a < 3; ++a) {
        ks.N[a] = p.grid[a];
        ks.kgrad[a] = c->tables + (size_t)a * 4096;
        ks.ufac[a] = c->tables + (size_t)(3 + a) * 4096;
        ks.eel[a] = c->tables + (size_t)(6 + a) * 4096;
        ks.k2[a] = c->tables + (size_t)(9 + a) * 4096;
    }
    ks.has_el = p.bjerrum > 0.0 ? 1 : 0;
    ks.sigma2 = (float)sigma2;
    ks.aq2 = (float)(p.a_charge * p.a_charge);
    for (int I = 0; I < S; ++I)
        for (int J = 0; J < S; ++J) {
            const double cij = (I == J) ? p.kappa / rho0 : (p.kappa + p.chi[I * TILD_MAX_SPECIES + J]) / rho0;  // A9
            ks.c[I * TILD_MAX_SPECIES + J] = (float)cij;
            ks.qq[I * TILD_MAX_SPECIES + J] = (float)(p.charge[I] * p.charge[J]);
        }

    // GJF constants (A11)
    StepParams& s = c->stp;
    const double gh = p.gamma * p.dt / (2.0 * p.mass);
    const double bg = 1.0 / (1.0 + gh), ag = (1.0 - gh) / (1.0 + gh);
    s.half_dt_over_m = (float)(p.dt / (2.0 * p.mass));
    s.kick_in = s.half_dt_over_m;
    s.a_g = (float)ag;
    s.w_fr = s.half_dt_over_m;
    s.b_dt = (float)(bg * p.dt);
    s.b_dt2_over_2m = (float)(bg * p.dt * p.dt / (2.0 * p.mass));
    s.b_dt_over_2m = (float)(bg * p.dt / (2.0 * p.mass));
    s.b_over_m = (float)(bg / p.mass);
    if (p.integrator == TILD_INTEGRATOR_VV) {   // velocity Verlet + Langevin ExtraForce (A24), c = 1 - gamma dt/2m
        const double cc = 1.0 - gh;
        s.a_g = (float)(cc * cc);
        s.w_fr = (float)(p.dt / (2.0 * p.mass * cc));
        s.b_dt = (float)(cc * p.dt);
        s.b_dt2_over_2m = (float)(p.dt * p.dt / (2.0 * p.mass));
        s.b_dt_over_2m = (float)(p.dt / (2.0 * p.mass));
        s.b_over_m = (float)((1.0 + cc) / (2.0 * p.mass));
    }
    s.dim2 = (p.flags & TILD_FLAG_2D) ? 1 : 0;
    s.noise_amp = (float)sqrt(2.0 * p.gamma * p.kT * p.dt);
    s.k_bond = (float)p.k_bond;
    s.r0_bond = (float)p.r0_bond;
    s.max_bonds = p.max_bonds;
    s.lambda_wlc = (p.max_bonds == 2) ? (float)p.lambda_wlc : 0.0f;
    s.k_theta = (p.max_bonds == 2) ? (float)p.k_theta : 0.0f;
    s.theta0 = (float)p.theta0;
    s.integrator = p.integrator;
    s.em_drift = p.gamma > 0.0 ? (float)(p.dt / p.gamma) : 0.0f;
    s.em_noise = p.gamma > 0.0 ? (float)(1.0 / p.gamma) : 0.0f;
    s.key0 = (uint32_t)(p.seed & 0xffffffffu);
    s.key1 = (uint32_t)(p.seed >> 32);

    cudaError_t e = cudaMemsetAsync(c->drift_count, 0, 4 * sizeof(uint32_t), c->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(c->tables, tab.data(), tab.size() * sizeof(float), cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);  // tab is a stack-owned host buffer
    if (e != cudaSuccess) {
        delete c;
        return TILD_ECUDA;
    }
    int dims[3] = {p.grid[0], p.grid[1], p.grid[2]};
    cufftHandle* plans[4] = {&c->plan_r2c, &c->plan_c2r, &c->plan_r2c_yz, &c->plan_c2r_yz};
    bool made[4] = {false, false, false, false};
    cufftResult fr = cufftPlanMany(&c->plan_r2c, 3, dims, nullptr, 1, 0, nullptr, 1, 0, CUFFT_R2C, S);
    made[0] = fr == CUFFT_SUCCESS;
    if (fr == CUFFT_SUCCESS && !c->xfft_R) {
        fr = cufftPlanMany(&c->plan_c2r, 3, dims, nullptr, 1, 0, nullptr, 1, 0, CUFFT_C2R, 3 * S);
        made[1] = fr == CUFFT_SUCCESS;
    }
    if (fr == CUFFT_SUCCESS && c->xfft_R) {   // contiguous (y, z) planes: batch = planes of all species / components
        fr = cufftPlanMany(&c->plan_r2c_yz, 2, dims + 1, nullptr, 1, 0, nullptr, 1, 0, CUFFT_R2C, S * p.grid[0]);
        made[2] = fr == CUFFT_SUCCESS;
        if (fr == CUFFT_SUCCESS) {
            fr = cufftPlanMany(&c->plan_c2r_yz, 2, dims + 1, nullptr, 1, 0, nullptr, 1, 0, CUFFT_C2R, 3 * S * p.grid[0]);
            made[3] = fr == CUFFT_SUCCESS;
        }
    }
    auto drop_plans = [&]() {
        for (int i = 0; i < 4; ++i)
            if (made[i]) cufftDestroy(*plans[i]);
    };
    if (fr != CUFFT_SUCCESS) {
        drop_plans();
        delete c;
        return TILD_ECUFFT;
    }
    if (fr == CUFFT_SUCCESS && (p.flags & TILD_FLAG_EXTRAS)) {
        fr = cufftPlanMany(&c->plan_x_r2c, 3, dims, nullptr, 1, 0, nullptr, 1, 0, CUFFT_R2C, 1);
        if (fr == CUFFT_SUCCESS) {
            fr = cufftPlanMany(&c->plan_x_c2r, 3, dims, nullptr, 1, 0, nullptr, 1, 0, CUFFT_C2R, 1);
            if (fr != CUFFT_SUCCESS) cufftDestroy(c->plan_x_r2c);
        }
        if (fr == CUFFT_SUCCESS) {
            c->xplans_ok = true;
            cufftSetStream(c->plan_x_r2c, c->stream);
            cufftSetStream(c->plan_x_c2r, c->stream);
        } else {
            drop_plans();
            delete c;
            return TILD_ECUFFT;
        }
    }
    if ((rc = tild_spread_configure(c)) != TILD_OK || (rc = tild_interp_configure(c)) != TILD_OK ||
        (rc = tild_kspace_configure(c)) != TILD_OK) {
        drop_plans();
        delete c;
        return rc;
    }
    c->plans_ok = true;
    for (int i = 0; i < 4; ++i)
        if (made[i]) cufftSetStream(*plans[i], c->stream);
    if (p.flags & TILD_FLAG_TIMING) {
        cudaError_t ee = cudaSuccess;
        int made_ev = 0;
        for (int i = 0; i < TILD_MAX_TIMED_STEPS && ee == cudaSuccess; ++i)
            for (int k = 0; k < TILD_N_STAGE_EVENTS && ee == cudaSuccess; ++k) {
                ee = cudaEventCreate(&c->ev[i][k]);
                if (ee == cudaSuccess) ++made_ev;
            }
        if (ee != cudaSuccess) {
            for (int j = 0; j < made_ev; ++j) cudaEventDestroy(c->ev[j / TILD_N_STAGE_EVENTS][j % TILD_N_STAGE_EVENTS]);
            drop_plans();
            delete c;
            return TILD_ECUDA;
        }
        c->ev_ok = true;
    }
    *out = c;
    return TILD_OK;
}

void tild_destroy(tild_ctx* c)
{
    if (!c) return;
    DevGuard dg(c);
    if (c->plans_ok) {
        cufftDestroy(c->plan_r2c);
        if (c->xfft_R) {
            cufftDestroy(c->plan_r2c_yz);
            cufftDestroy(c->plan_c2r_yz);
        } else {
            cufftDestroy(c->plan_c2r);
        }
    }
    if (c->xplans_ok) {
        cufftDestroy(c->plan_x_r2c);
        cufftDestroy(c->plan_x_c2r);
    }
    drop_graphs(c);
    if (c->hp_in) {
        cudaStreamSynchronize(c->hp_in);
        cudaStreamSynchronize(c->hp_out);
        cudaEventDestroy(c->hp_ev_in);
        cudaEventDestroy(c->hp_ev_done);
        for (int k = 0; k < 4; ++k) cudaEventDestroy(c->hp_ev_out[k]);
        cudaStreamDestroy(c->hp_in);
        cudaStreamDestroy(c->hp_out);
    }
    if (c->copy_stream) {
        cudaStreamSynchronize(c->copy_stream);
        for (int k = 0; k < 2; ++k)
            if (c->copy_ev[k]) cudaEventDestroy(c->copy_ev[k]);
        cudaStreamDestroy(c->copy_stream);
    }
    if (c->ev_ok)
        for (int i = 0; i < TILD_MAX_TIMED_STEPS; ++i)
            for (int k = 0; k < TILD_N_STAGE_EVENTS; ++k) cudaEventDestroy(c->ev[i][k]);
    delete c;
}

const char* tild_last_error(const tild_ctx* c) { return c ? c->err : "null context"; }
int64_t tild_launch_count(const tild_ctx* c) { return c ? c->launches : 0; }

int tild_layout_info(const tild_ctx* c, uint64_t info[8])
{
    if (!c || !info) return TILD_EINVAL;
    if (!c->has_state) return TILD_ESTATE;
    const TileParams& t = c->tile;
    const uint64_t v[8] = {(uint64_t)t.ntiles, (uint64_t)t.nseg, (uint64_t)t.EZ, (uint64_t)t.smem_spread, (uint64_t)t.smem_interp,
                           (uint64_t)t.T[0], (uint64_t)t.T[1], (uint64_t)t.T[2]};
    for (int k = 0; k < 8; ++k) info[k] = v[k];
    return TILD_OK;
}

int tild_segment_layout(const tild_ctx* cc, uint32_t* seg_base, uint32_t* slot_id)
{
    tild_ctx* c = const_cast<tild_ctx*>(cc);
    if (!c) return TILD_EINVAL;
    DevGuard dg(c);
    if (!c->has_state) return tild_fail(c, TILD_ESTATE, "tild_segment_layout before tild_set_state");
    if (seg_base)
        TILD_CUDA(c, cudaMemcpyAsync(seg_base, c->lay.seg_base, ((size_t)c->tile.nseg + 1) * sizeof(uint32_t), cudaMemcpyDeviceToDevice, c->stream));
    if (slot_id) return launch_slot_ids(c, slot_id);
    return TILD_OK;
}

int tild_spread(tild_ctx* c, const float* x, const int32_t* type, float* grid)
{
    DevGuard dg(c);
    if (!c || !grid || (c->mesh.n > 0 && (!x || !type))) return tild_fail(c, TILD_EINVAL, "tild_spread: null argument");
    int rc = stage_layout(c, x, type);  // slab-ordered copy of the caller's particles
    if (rc) return rc;
    return launch_spread(c, c->lay_stage, c->SX4, grid);
}

int tild_kspace_force(tild_ctx* c, const float* grid, float* ffield)
{
    DevGuard dg(c);
    if (!c || !grid || !ffield) return tild_fail(c, TILD_EINVAL, "tild_kspace_force: null argument");
    return kspace_pipeline(c, grid, ffield, nullptr);
}

int tild_interp(tild_ctx* c, const float* ffield, const float* x, const int32_t* type, float* f)
{
    DevGuard dg(c);
    if (!c || !ffield || (c->mesh.n > 0 && (!x || !type || !f))) return tild_fail(c, TILD_EINVAL, "tild_interp: null argument");
    const int n = c->mesh.n;
    if (n == 0) return TILD_OK;
    int rc = stage_layout(c, x, type);
    if (rc) return rc;
    rc = launch_interp(c, INTERP_NONBONDED_BY_ID, c->lay_stage, ffield, c->SX4, nullptr, nullptr, nullptr, nullptr, nullptr);
    if (rc) return rc;
    gather_by_inv_kernel<<<(n + 255) / 256, 256, 0, c->stream>>>(n, c->inv, c->F4, f);
    TILD_LAUNCH_CHECK(c, "gather_by_inv_kernel");
    return TILD_OK;
}

int tild_bond_force(tild_ctx* c, const float* x, const int32_t* bond_partner, float* f)
{
    DevGuard dg(c);
    if (!c || (c->mesh.n > 0 && (!x || !f))) return tild_fail(c, TILD_EINVAL, "tild_bond_force: null argument");
    if (c->stp.max_bonds > 0 && !bond_partner && c->mesh.n > 0) return tild_fail(c, TILD_EINVAL, "tild_bond_force: null partners");
    return launch_bond_force_caller(c, x, bond_partner, f);
}

int tild_index_map(tild_ctx* c, const float* x, int32_t* base, uint32_t* cell_key, uint32_t* perm, uint32_t* cell_start)
{
    DevGuard dg(c);
    if (!c || (c->mesh.n > 0 && !x)) return tild_fail(c, TILD_EINVAL, "tild_index_map: null argument");
    uint32_t* key = cell_key ? cell_key : c->key;
    int rc = launch_cell_keys(c, x, key, base);
    if (rc) return rc;
    if (perm || cell_start) rc = launch_counting_sort(c, key, c->M, perm ? perm : c->perm, cell_start ? cell_start : c->start);
    return rc;
}

int tild_philox_test(tild_ctx* c, const uint32_t* ctr, const uint32_t* key, uint32_t* out, float* gauss, int32_t m)
{
    DevGuard dg(c);
    if (!c || (m > 0 && (!ctr || !key || !out))) return tild_fail(c, TILD_EINVAL, "tild_philox_test: null argument");
    return launch_philox_test(c, ctr, key, out, gauss, m);
}

int tild_set_state(tild_ctx* c, const float* x, const float* v, const int32_t* type, const int32_t* bond_partner, uint64_t step0)
{
    DevGuard dg(c);
    if (!c) return TILD_EINVAL;
    const size_t n = (size_t)c->mesh.n;
    if (n > 0 && (!x || !v || !type)) return tild_fail(c, TILD_EINVAL, "tild_set_state: null argument");
    if (n > 0 && c->stp.max_bonds > 0 && !bond_partner) return tild_fail(c, TILD_EINVAL, "tild_set_state: null bond_partner");
    c->cur = 0;
    c->lay_valid = false;                       // the first sort of a state has no order to keep
    c->has_state = false;
    TILD_CUDA(c, cudaMemsetAsync(c->drift_count, 0, 4 * sizeof(uint32_t), c->stream));
    int rc = launch_pack(c, x, v, type, c->stp.max_bonds > 0 ? bond_partner : nullptr, c->X4[0], c->W4[0], c->B[0]);
    if (rc) return rc;
    if (n > 0) {   // argument check (include/tild.h): one 4-byte read-back and a synchronisation per tild_set_state
        uint32_t bad = 0;
        TILD_CUDA(c, cudaMemcpyAsync(&bad, c->drift_count + 2, sizeof(uint32_t), cudaMemcpyDeviceToHost, c->stream));
        TILD_CUDA(c, cudaStreamSynchronize(c->stream));
        if (bad) return tild_fail(c, TILD_EINVAL, "tild_set_state: a type is outside [0, %d) or a bond partner outside [-1, %d)", c->mesh.S, c->mesh.n);
    }
    if ((rc = launch_reorder(c))) return rc;
    c->resorts_since_defrag = 0;
    // The state array holds v itself until the first step: that step takes v^0 as it is (kick_in = 0) and leaves the
    // split-kick state w^1 = v^1 - (dt/2m) F^1 behind, so loading a state costs a sort and no force evaluation.
    c->stp.kick_in = 0.0f;
    c->step = step0;
    c->h_step_upload = step0;
    TILD_CUDA(c, cudaMemcpyAsync(c->d_step, &c->h_step_upload, sizeof(uint64_t), cudaMemcpyHostToDevice, c->stream));
    c->has_state = true;
    c->timed_steps = 0;
    c->ms_steps = 0;
    for (int k = 0; k < 8; ++k) c->ms_sum[k] = 0.0;
    return TILD_OK;
}

}  // extern "C"

namespace {

// Synchronises and adds the recorded stage events of the last `timed_steps` steps to the running sums, so that the
// event ring (TILD_MAX_TIMED_STEPS steps) never limits how many steps are timed.
int fold_timings(tild_ctx* c)
{
    if (!c->ev_ok || c->timed_steps == 0) return TILD_OK;
    TILD_CUDA(c, cudaStreamSynchronize(c->stream));
    for (int i = 0; i < c->timed_steps; ++i) {
        for (int k = 0; k < 6; ++k) {
            float t = 0.0f;
            TILD_CUDA(c, cudaEventElapsedTime(&t, c->ev[i][k], c->ev[i][k + 1]));
            c->ms_sum[k] += t;
        }
        float tot = 0.0f;
        TILD_CUDA(c, cudaEventElapsedTime(&tot, c->ev[i][0], c->ev[i][6]));
        c->ms_sum[7] += tot;
    }
    c->ms_steps += c->timed_steps;
    c->timed_steps = 0;
    return TILD_OK;
}

// one TILD step on the internal state (re-sort when due, mesh pipeline, fused interpolation pass, step counter)
int enqueue_one_step(tild_ctx* c, cudaEvent_t* ev, bool allow_defrag)
{
    if (ev) TILD_CUDA(c, cudaEventRecord(ev[0], c->stream));
    if (c->steps_since_sort >= c->resort_every) {
        const bool defrag = allow_defrag && c->resorts_since_defrag >= TILD_DEFRAG_EVERY && !(c->prm.flags & TILD_FLAG_NO_DEFRAG) &&
                            (c->mesh.n >= TILD_DEFRAG_MIN_N || (c->prm.flags & TILD_FLAG_DEFRAG_SMALL));
        int rc = defrag ? launch_defrag(c) : launch_reorder(c);
        if (rc) return rc;
    }
    if (ev) TILD_CUDA(c, cudaEventRecord(ev[1], c->stream));
    const int a = c->cur;
    int rc = mesh_pipeline(c, c->lay, c->X4[a], ev);
    if (rc) return rc;
    if ((rc = launch_extra_forces(c, c->X4[a], c->W4[a]))) return rc;   // per-particle charges / Maier-Saupe -> Fext
    rc = launch_interp(c, INTERP_FUSED_STEP, c->lay, c->ffield, c->X4[a], c->W4[a], c->B[a], c->X4[1 - a], c->W4[1 - a], nullptr);
    if (rc) return rc;
    if ((rc = launch_extra_apply(c, 2, c->stp.kick_in, c->X4[1 - a], c->W4[1 - a]))) return rc;
    // from here on the state is w = v - (dt/2m) F (Euler-Maruyama never touches the velocities: the state stays v)
    c->stp.kick_in = c->stp.integrator == TILD_INTEGRATOR_EM ? 0.0f : c->stp.half_dt_over_m;
    if (!c->step_advanced && (rc = launch_advance_step(c))) return rc;   // per-particle path: no drift kernel to do it
    // swap only the x/w pointers so that `cur` keeps naming the buffer that holds the bond table
    float4* t = c->X4[a]; c->X4[a] = c->X4[1 - a]; c->X4[1 - a] = t;
    t = c->W4[a]; c->W4[a] = c->W4[1 - a]; c->W4[1 - a] = t;
    if (ev) TILD_CUDA(c, cudaEventRecord(ev[6], c->stream));
    c->step++;
    c->steps_since_sort++;
    return TILD_OK;
}

// Graph replay.  Block 0: two re-sort cycles (2 * resort_every steps, starting with a re-sort).  After an even number of
// steps per cycle and two cycles every buffer pointer is back where it started, and the step index lives in device
// memory, so the instantiated graph can be replayed as it is.  Block 1 (with_defrag): ONE cycle that starts with the return
// to particle-id order -- launch_defrag flips the buffers twice (to id order, then the sort), so one cycle already ends where
// it started; without it the step at which the return is due and the rest of its cycle ran as single launches.
int launch_graph_block(tild_ctx* c, bool with_defrag)
{
    const int g = with_defrag ? 1 : 0;
    const int block = (with_defrag ? 1 : 2) * c->resort_every;
    if (!c->grid_clean) {   // the captured block starts from a cleared density grid (its steps clear it for one another)
        TILD_CUDA(c, cudaMemsetAsync(c->grid, 0, sizeof(float) * c->M * c->mesh.S, c->stream));
        c->grid_clean = true;
    }
    if (!(c->graph_ok[g] && c->graph_cur[g] == c->cur && c->graph_x0[g] == c->X4[0])) {
        if (c->graph_ok[g]) {
            cudaGraphExecDestroy(c->graph_exec[g]);
            c->graph_ok[g] = false;
        }
        // capture: nothing executes, so the host bookkeeping the enqueue advances is put back afterwards
        const int cur0 = c->cur, sss0 = c->steps_since_sort, rsd0 = c->resorts_since_defrag;
        const bool lay_valid0 = c->lay_valid;
        const uint64_t step0 = c->step;
        const int64_t launches0 = c->launches;
        float4* const x0[2] = {c->X4[0], c->X4[1]};
        float4* const w0[2] = {c->W4[0], c->W4[1]};
        TILD_CUDA(c, cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeThreadLocal));
        int rc = TILD_OK;
        for (int i = 0; i < block && rc == TILD_OK; ++i) rc = enqueue_one_step(c, nullptr, with_defrag && i == 0);
        cudaGraph_t graph = nullptr;
        const cudaError_t e = cudaStreamEndCapture(c->stream, &graph);
        c->graph_launches[g] = c->launches - launches0;
        c->graph_leaves_clean2[g] = c->grid_clean;
        c->grid_clean = true;   // nothing ran
        const bool same = c->cur == cur0 && c->X4[0] == x0[0] && c->W4[0] == w0[0] && c->steps_since_sort == sss0;
        c->cur = cur0; c->steps_since_sort = sss0; c->step = step0; c->launches = launches0; c->resorts_since_defrag = rsd0;
        c->lay_valid = lay_valid0;
        c->X4[0] = x0[0]; c->X4[1] = x0[1]; c->W4[0] = w0[0]; c->W4[1] = w0[1];
        if (rc != TILD_OK || e != cudaSuccess || !graph || !same) {
            if (graph) cudaGraphDestroy(graph);
            if (rc != TILD_OK) return rc;
            return tild_fail(c, TILD_ECUDA, "CUDA graph capture of %d steps failed: %s", block,
                             e != cudaSuccess ? cudaGetErrorString(e) : "state does not return to its start");
        }
        const cudaError_t ei = cudaGraphInstantiate(&c->graph_exec[g], graph, 0);
        cudaGraphDestroy(graph);
        if (ei != cudaSuccess) return tild_fail(c, TILD_ECUDA, "cudaGraphInstantiate: %s", cudaGetErrorString(ei));
        c->graph_ok[g] = true;
        c->graph_cur[g] = c->cur;
        c->graph_x0[g] = c->X4[0];
    }
    TILD_CUDA(c, cudaGraphLaunch(c->graph_exec[g], c->stream));
    c->grid_clean = c->graph_leaves_clean2[g];
    c->step += (uint64_t)block;          // pointers, cur and steps_since_sort end where they started
    if (with_defrag) {
        c->resorts_since_defrag = 0;
        c->lay_valid = true;             // the sort inside the block was the sort of a fresh state: c->lay describes X4[cur]
    } else {
        c->resorts_since_defrag += 2;
    }
    c->launches += c->graph_launches[g];
    return TILD_OK;
}

}  // namespace

extern "C" {

int tild_step(tild_ctx* c, int32_t nsteps)
{
    DevGuard dg(c);
    if (!c) return TILD_EINVAL;
    if (!c->has_state) return tild_fail(c, TILD_ESTATE, "tild_step before tild_set_state");
    if (nsteps < 0) return tild_fail(c, TILD_EINVAL, "tild_step: nsteps < 0");
    // stream capture is not available on the legacy default stream (NULL / cudaStreamLegacy)
    const bool graphs = !(c->prm.flags & TILD_FLAG_EAGER) && !c->ev_ok && c->resort_every % 2 == 0 && c->stream != nullptr &&
                        c->stream != cudaStreamLegacy;
    int32_t s = 0;
    while (s < nsteps) {
        // a return to particle-id order that is due takes the place of the re-sort that starts a cycle: as a captured block of
        // one cycle where graphs replay, as the re-sort of an eager step otherwise
        const bool defrag_due = c->steps_since_sort >= c->resort_every && c->resorts_since_defrag >= TILD_DEFRAG_EVERY &&
                                !(c->prm.flags & TILD_FLAG_NO_DEFRAG) && (c->mesh.n >= TILD_DEFRAG_MIN_N || (c->prm.flags & TILD_FLAG_DEFRAG_SMALL));
        if (graphs && c->steps_since_sort >= c->resort_every && nsteps - s >= (defrag_due ? 1 : 2) * c->resort_every) {
            int rc = launch_graph_block(c, defrag_due);
            if (rc) return rc;
            s += (defrag_due ? 1 : 2) * c->resort_every;
            continue;
        }
        if (c->ev_ok && c->timed_steps == TILD_MAX_TIMED_STEPS) {   // ring full: fold it into the sums (synchronises)
            int rcf = fold_timings(c);
            if (rcf) return rcf;
        }
        cudaEvent_t* ev = c->ev_ok ? c->ev[c->timed_steps] : nullptr;
        int rc = enqueue_one_step(c, ev, true);
        if (rc) return rc;
        if (ev) c->timed_steps++;
        ++s;
    }
    return TILD_OK;
}

int tild_get_state(tild_ctx* c, float* x, float* v, float* f, uint64_t* step)
{
    DevGuard dg(c);
    if (!c) return TILD_EINVAL;
    if (!c->has_state) return tild_fail(c, TILD_ESTATE, "tild_get_state before tild_set_state");
    const size_t n = (size_t)c->mesh.n;
    const size_t bytes = 3 * n * sizeof(float);
    if (step) *step = c->step;
    if (n == 0) return TILD_OK;
    const int a = c->cur;
    float* scratch = reinterpret_cast<float*>(c->SX4);  // [n][3] staging in caller order; x/v/f may be host pointers
    int rc;
    const bool need_force = f || (v && c->stp.kick_in != 0.0f);   // v = w + (dt/2m) F needs F(x); right after tild_set_state the state is v itself
    bool x_in_flight = false;
    if (x) {
        if ((rc = launch_unpermute(c, c->X4[a], scratch))) return rc;
        // large systems: the copy of x (PCIe when x is a host pointer) runs on a second stream under the force evaluation
        if (need_force && n >= (size_t)1 << 18 && c->stream != nullptr && c->stream != cudaStreamLegacy) {
            if (!c->copy_stream) {
                TILD_CUDA(c, cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking));
                for (int k = 0; k < 2; ++k) TILD_CUDA(c, cudaEventCreateWithFlags(&c->copy_ev[k], cudaEventDisableTiming));
            }
            TILD_CUDA(c, cudaEventRecord(c->copy_ev[0], c->stream));
            TILD_CUDA(c, cudaStreamWaitEvent(c->copy_stream, c->copy_ev[0], 0));
            TILD_CUDA(c, cudaMemcpyAsync(x, scratch, bytes, cudaMemcpyDefault, c->copy_stream));
            TILD_CUDA(c, cudaEventRecord(c->copy_ev[1], c->copy_stream));
            x_in_flight = true;
        } else {
            TILD_CUDA(c, cudaMemcpyAsync(x, scratch, bytes, cudaMemcpyDefault, c->stream));
        }
    }
    if (need_force) rc = force_current(c);
    if (x_in_flight) TILD_CUDA(c, cudaStreamWaitEvent(c->stream, c->copy_ev[1], 0));   // scratch is reused below; stream order for the caller
    if (rc) return rc;
    if (v || f) {
        if (f) {
            if ((rc = launch_unpermute(c, c->F4, scratch))) return rc;
            TILD_CUDA(c, cudaMemcpyAsync(f, scratch, bytes, cudaMemcpyDefault, c->stream));
        }
        if (v) {
            if ((rc = launch_velocity_out(c, c->F4, c->W4[a], scratch))) return rc;  // v = w + (dt/2m) F
            TILD_CUDA(c, cudaMemcpyAsync(v, scratch, bytes, cudaMemcpyDefault, c->stream));
        }
    }
    return TILD_OK;
}

int tild_energy(tild_ctx* c, double e[3])
{
    DevGuard dg(c);
    if (!c || !e) return TILD_EINVAL;
    if (!c->has_state) return tild_fail(c, TILD_ESTATE, "tild_energy before tild_set_state");
    int rc = force_current(c);              // F4 and nhat at the current positions; no state change
    if (rc) return rc;
    if (c->xfft_R)   // the fused x-transform leaves nhat transformed over (y, z) only: redo the full transform of the densities
        TILD_FFT(c, cufftExecR2C(c->plan_r2c, c->grid, reinterpret_cast<cufftComplex*>(c->nhat)));
    if ((rc = launch_energy(c, c->d_energy))) return rc;
    TILD_CUDA(c, cudaMemcpyAsync(e, c->d_energy, 3 * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    TILD_CUDA(c, cudaStreamSynchronize(c->stream));
    return TILD_OK;
}

int tild_set_charges(tild_ctx* c, const float* q)
{
    DevGuard dg(c);
    if (!c) return TILD_EINVAL;
    if (!c->Fext) return tild_fail(c, TILD_EINVAL, "tild_set_charges needs TILD_FLAG_EXTRAS at tild_init");
    c->has_q = q != nullptr;
    c->ksp.has_el = (c->prm.bjerrum > 0.0 && !c->has_q) ? 1 : 0;     // A25: the charge mesh replaces the charges per species
    drop_graphs(c);                                                  // a captured block has the old choice baked in
    if (q && c->mesh.n > 0)
        TILD_CUDA(c, cudaMemcpyAsync(c->q_id, q, sizeof(float) * (size_t)c->mesh.n, cudaMemcpyDeviceToDevice, c->stream));
    return TILD_OK;
}

int tild_set_ms_partners(tild_ctx* c, const int32_t* partner)
{
    DevGuard dg(c);
    if (!c) return TILD_EINVAL;
    if (!c->Fext) return tild_fail(c, TILD_EINVAL, "tild_set_ms_partners needs TILD_FLAG_EXTRAS at tild_init");
    c->has_ms = partner != nullptr;
    drop_graphs(c);                                                  // a captured block has the old choice baked in
    if (partner && c->mesh.n > 0)
        TILD_CUDA(c, cudaMemcpyAsync(c->msp_id, partner, sizeof(int32_t) * (size_t)c->mesh.n, cudaMemcpyDeviceToDevice, c->stream));
    return TILD_OK;
}

int tild_virial(tild_ctx* c, double w[2])
{
    DevGuard dg(c);
    if (!c || !w) return TILD_EINVAL;
    double e[3];
    int rc = tild_energy(c, e);             // fills d_energy[0..4]
    if (rc) return rc;
    TILD_CUDA(c, cudaMemcpyAsync(w, c->d_energy + 3, 2 * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    TILD_CUDA(c, cudaStreamSynchronize(c->stream));
    if (c->prm.flags & TILD_FLAG_SAMPLED_KERNEL) w[1] = NAN;   // k . grad u^ of the sampled kernel has no closed form
    return TILD_OK;
}

int tild_structure_factor(tild_ctx* c, uint32_t species_mask, float* sk, int32_t accumulate)
{
    DevGuard dg(c);
    if (!c || !sk) return tild_fail(c, TILD_EINVAL, "tild_structure_factor: null argument");
    if (!c->has_state) return tild_fail(c, TILD_ESTATE, "tild_structure_factor before tild_set_state");
    if ((species_mask & ((1u << c->mesh.S) - 1u)) == 0) return tild_fail(c, TILD_EINVAL, "tild_structure_factor: empty species mask");
    int rc = launch_spread(c, c->lay, c->X4[c->cur], c->grid);
    if (rc) return rc;
    TILD_FFT(c, cufftExecR2C(c->plan_r2c, c->grid, reinterpret_cast<cufftComplex*>(c->nhat)));
    return launch_structure_factor(c, species_mask, sk, accumulate);
}

int tild_get_timings(tild_ctx* c, float ms[8], int32_t* steps_timed)
{
    DevGuard dg(c);
    if (!c || !ms) return TILD_EINVAL;
    for (int k = 0; k < 8; ++k) ms[k] = 0.0f;
    if (steps_timed) *steps_timed = 0;
    TILD_CUDA(c, cudaStreamSynchronize(c->stream));
    int rc = fold_timings(c);
    if (rc) return rc;
    if (!c->ev_ok || c->ms_steps == 0) return TILD_OK;
    const double T = (double)c->ms_steps;
    for (int k = 0; k < 8; ++k) ms[k] = (float)(c->ms_sum[k] / T);
    ms[6] = ms[7] - (ms[0] + ms[1] + ms[2] + ms[3] + ms[4] + ms[5]);
    if (steps_timed) *steps_timed = (int32_t)c->ms_steps;
    for (int k = 0; k < 8; ++k) c->ms_sum[k] = 0.0;
    c->ms_steps = 0;
    c->timed_steps = 0;
    return TILD_OK;
}

int tild_run_host(tild_ctx* c, float* x_host, float* v_host, const int32_t* type_host, const int32_t* bond_partner_host,
                  uint64_t step0, int32_t nsteps)
{
    DevGuard dg(c);
    if (!c) return TILD_EINVAL;
    const size_t n = (size_t)c->mesh.n;
    const size_t mb = (size_t)c->stp.max_bonds;
    if (n > 0 && (!x_host || !v_host || !type_host || (mb > 0 && !bond_partner_host)))
        return tild_fail(c, TILD_EINVAL, "tild_run_host: null argument");
    // device staging of the host batch in scratch that tild_set_state only touches after it has packed the batch
    float* xs = reinterpret_cast<float*>(c->SX4);
    float* vs = reinterpret_cast<float*>(c->F4);
    int32_t* ts = reinterpret_cast<int32_t*>(c->key);
    int32_t* bs = c->B[1];
    if (n > 0) {
        TILD_CUDA(c, cudaMemcpyAsync(xs, x_host, 3 * n * sizeof(float), cudaMemcpyHostToDevice, c->stream));
        TILD_CUDA(c, cudaMemcpyAsync(vs, v_host, 3 * n * sizeof(float), cudaMemcpyHostToDevice, c->stream));
        TILD_CUDA(c, cudaMemcpyAsync(ts, type_host, n * sizeof(int32_t), cudaMemcpyHostToDevice, c->stream));
        if (mb > 0) TILD_CUDA(c, cudaMemcpyAsync(bs, bond_partner_host, n * mb * sizeof(int32_t), cudaMemcpyHostToDevice, c->stream));
    }
    int rc = tild_set_state(c, xs, vs, ts, bs, step0);
    if (rc) return rc;
    if ((rc = tild_step(c, nsteps))) return rc;
    if ((rc = tild_get_state(c, x_host, v_host, nullptr, nullptr))) return rc;
    TILD_CUDA(c, cudaStreamSynchronize(c->stream));
    return TILD_OK;
}

// Pipelined end-to-end path for independent batches: the copy of batch k + 1 to the device and the copy of batch k - 1 to
// the host run on their own streams under the computation of batch k (PCIe is full duplex; C4 moves 302 MB in and 201 MB
// out per batch, three times the time of the kernels).
int tild_run_host_submit(tild_ctx* c, const float* x_host, const float* v_host, const int32_t* type_host, const int32_t* bond_partner_host,
                         uint64_t step0, int32_t nsteps, float* x_out_host, float* v_out_host)
{
    DevGuard dg(c);
    if (!c) return TILD_EINVAL;
    if (!c->hp_xo[0]) return tild_fail(c, TILD_EINVAL, "tild_run_host_submit needs TILD_FLAG_HOST_PIPELINE at tild_init");
    const size_t n = (size_t)c->mesh.n, mb = (size_t)c->stp.max_bonds;
    if (n > 0 && (!x_host || !v_host || !type_host || (mb > 0 && !bond_partner_host) || !x_out_host || !v_out_host))
        return tild_fail(c, TILD_EINVAL, "tild_run_host_submit: null argument");
    if (c->stream == nullptr || c->stream == cudaStreamLegacy)
        return tild_fail(c, TILD_EINVAL, "tild_run_host_submit needs a context on a stream of its own (the legacy default stream synchronises with every other stream)");
    if (!c->hp_in) {
        TILD_CUDA(c, cudaStreamCreateWithFlags(&c->hp_in, cudaStreamNonBlocking));
        TILD_CUDA(c, cudaStreamCreateWithFlags(&c->hp_out, cudaStreamNonBlocking));
        TILD_CUDA(c, cudaEventCreateWithFlags(&c->hp_ev_in, cudaEventDisableTiming));
        TILD_CUDA(c, cudaEventCreateWithFlags(&c->hp_ev_done, cudaEventDisableTiming));
        for (int k = 0; k < 4; ++k) TILD_CUDA(c, cudaEventCreateWithFlags(&c->hp_ev_out[k], cudaEventDisableTiming));
    }
    if (c->hp_submitted - c->hp_waited >= 4)
        return tild_fail(c, TILD_ESTATE, "tild_run_host_submit: four batches in flight, call tild_run_host_wait first");
    const int slot = (int)(c->hp_submitted & 1u), ev = (int)(c->hp_submitted & 3u);
    if (n > 0) {
        // the input staging is free: the tild_set_state of the previous submit synchronised after packing it
        TILD_CUDA(c, cudaMemcpyAsync(c->hp_x, x_host, 3 * n * sizeof(float), cudaMemcpyHostToDevice, c->hp_in));
        TILD_CUDA(c, cudaMemcpyAsync(c->hp_v, v_host, 3 * n * sizeof(float), cudaMemcpyHostToDevice, c->hp_in));
        TILD_CUDA(c, cudaMemcpyAsync(c->hp_t, type_host, n * sizeof(int32_t), cudaMemcpyHostToDevice, c->hp_in));
        if (mb > 0) TILD_CUDA(c, cudaMemcpyAsync(c->hp_b, bond_partner_host, n * mb * sizeof(int32_t), cudaMemcpyHostToDevice, c->hp_in));
    }
    TILD_CUDA(c, cudaEventRecord(c->hp_ev_in, c->hp_in));
    TILD_CUDA(c, cudaStreamWaitEvent(c->stream, c->hp_ev_in, 0));
    int rc = tild_set_state(c, c->hp_x, c->hp_v, c->hp_t, c->hp_b, step0);   // synchronises: the staging is consumed
    if (rc) return rc;
    if ((rc = tild_step(c, nsteps))) return rc;
    if (c->hp_submitted >= 2) TILD_CUDA(c, cudaStreamWaitEvent(c->stream, c->hp_ev_out[(ev + 2) & 3], 0));   // batch k - 2 has left this output set
    if ((rc = tild_get_state(c, c->hp_xo[slot], c->hp_vo[slot], nullptr, nullptr))) return rc;
    TILD_CUDA(c, cudaEventRecord(c->hp_ev_done, c->stream));
    TILD_CUDA(c, cudaStreamWaitEvent(c->hp_out, c->hp_ev_done, 0));
    if (n > 0) {
        TILD_CUDA(c, cudaMemcpyAsync(x_out_host, c->hp_xo[slot], 3 * n * sizeof(float), cudaMemcpyDeviceToHost, c->hp_out));
        TILD_CUDA(c, cudaMemcpyAsync(v_out_host, c->hp_vo[slot], 3 * n * sizeof(float), cudaMemcpyDeviceToHost, c->hp_out));
    }
    TILD_CUDA(c, cudaEventRecord(c->hp_ev_out[ev], c->hp_out));
    c->hp_submitted++;
    return TILD_OK;
}

int tild_run_host_wait(tild_ctx* c)
{
    DevGuard dg(c);
    if (!c) return TILD_EINVAL;
    if (c->hp_waited >= c->hp_submitted) return tild_fail(c, TILD_ESTATE, "tild_run_host_wait: no batch in flight");
    TILD_CUDA(c, cudaEventSynchronize(c->hp_ev_out[c->hp_waited & 3u]));   // at most four in flight: the event is this batch's
    c->hp_waited++;
    return TILD_OK;
}

}  // extern "C"
