// a1: canonical fp32 index map, cell keys, counting sort by cell (the stage call tild_index_map),
// and the slab-transposed ("ELL") re-ordering of the internal particle state that the tile kernels run on.
// Not in the paper's PM text; nearest prior art is its neighbour-list cell binning with atomics
// (PAPER.md L205).  DESIGN.md A15/A16 define what is bit-exact; DESIGN.md section 4 describes the layout.
#include "tild_internal.cuh"

namespace {

constexpr int SCAN_THREADS = 256;
constexpr int SCAN_ITEMS = 16;
constexpr int SCAN_CHUNK = SCAN_THREADS * SCAN_ITEMS;  // 4096 elements per block

template <int P>
__global__ void __launch_bounds__(256) cell_key_kernel(MeshParams m, const float* __restrict__ x,
                                                       uint32_t* __restrict__ key, int32_t* __restrict__ base)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= m.n) return;
    int c[3], b[3];
    float t;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        index_1d<P>(x[3 * (size_t)i + a], m.inv_h[a], c[a], b[a], t);
        c[a] = wrap_idx(c[a], m.N[a]);
    }
    if (key) key[i] = (uint32_t)((c[0] * m.N[1] + c[1]) * m.N[2] + c[2]);
    if (base) {
        base[3 * (size_t)i + 0] = b[0];
        base[3 * (size_t)i + 1] = b[1];
        base[3 * (size_t)i + 2] = b[2];
    }
}

// count[key]++ ; rank[i] = arrival order inside the bin
__global__ void __launch_bounds__(256) histogram_kernel(int n, const uint32_t* __restrict__ key,
                                                        uint32_t* __restrict__ count, uint32_t* __restrict__ rank)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    rank[i] = atomicAdd(&count[key[i]], 1u);
}

__device__ __forceinline__ uint32_t warp_incl_scan(uint32_t v)
{
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const uint32_t o = __shfl_up_sync(0xffffffffu, v, d);
        if ((threadIdx.x & 31) >= d) v += o;
    }
    return v;
}

// exclusive scan of one value per thread across the block; returns the exclusive prefix, *total = block sum
template <int NT>
__device__ __forceinline__ uint32_t block_excl_scan(uint32_t v, uint32_t* total)
{
    __shared__ uint32_t warp_sums[NT / 32];
    __shared__ uint32_t block_total;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const uint32_t incl = warp_incl_scan(v);
    if (lane == 31) warp_sums[wid] = incl;
    __syncthreads();
    if (wid == 0) {
        uint32_t s = lane < NT / 32 ? warp_sums[lane] : 0u;
        const uint32_t si = warp_incl_scan(s);
        if (lane < NT / 32) warp_sums[lane] = si - s;
        if (lane == NT / 32 - 1) block_total = si;
    }
    __syncthreads();
    const uint32_t r = warp_sums[wid] + incl - v;
    if (total) *total = block_total;
    __syncthreads();
    return r;
}

__global__ void __launch_bounds__(SCAN_THREADS) scan_reduce_kernel(size_t len, const uint32_t* __restrict__ in,
                                                                   uint32_t* __restrict__ part)
{
    const size_t start = (size_t)blockIdx.x * SCAN_CHUNK;
    uint32_t s = 0;
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        const size_t j = start + (size_t)k * SCAN_THREADS + threadIdx.x;
        if (j < len) s += in[j];
    }
    uint32_t total;
    block_excl_scan<SCAN_THREADS>(s, &total);
    if (threadIdx.x == 0) part[blockIdx.x] = total;
}

// single block: exclusive scan of part[0..nb) in place
__global__ void __launch_bounds__(1024) scan_parts_kernel(int nb, uint32_t* __restrict__ part)
{
    const int per = (nb + 1023) / 1024;
    const int lo = threadIdx.x * per;
    uint32_t s = 0;
    for (int k = 0; k < per; ++k)
        if (lo + k < nb) s += part[lo + k];
    uint32_t run = block_excl_scan<1024>(s, nullptr);
    for (int k = 0; k < per; ++k)
        if (lo + k < nb) {
            const uint32_t v = part[lo + k];
            part[lo + k] = run;
            run += v;
        }
}

__global__ void __launch_bounds__(SCAN_THREADS) scan_final_kernel(size_t len, const uint32_t* __restrict__ in,
                                                                  const uint32_t* __restrict__ part,
                                                                  uint32_t* __restrict__ out)
{
    const size_t start = (size_t)blockIdx.x * SCAN_CHUNK + (size_t)threadIdx.x * SCAN_ITEMS;
    uint32_t v[SCAN_ITEMS];
    uint32_t s = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        v[k] = start + k < len ? in[start + k] : 0u;
        s += v[k];
    }
    uint32_t run = block_excl_scan<SCAN_THREADS>(s, nullptr) + part[blockIdx.x];
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        if (start + k < len) out[start + k] = run;
        run += v[k];
    }
}

// perm[cell_start[key] + rank] = i
__global__ void __launch_bounds__(256) scatter_perm_kernel(int n, const uint32_t* __restrict__ key,
                                                           const uint32_t* __restrict__ cell_start,
                                                           const uint32_t* __restrict__ rank, uint32_t* __restrict__ perm)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    perm[cell_start[key[i]] + rank[i]] = (uint32_t)i;
}

// ---- slab-transposed layout ---------------------------------------------------------------------------------------

// caller arrays -> slots [0, n): slot i holds particle id i
__global__ void __launch_bounds__(256) pack_kernel(int n, int max_bonds, const float* __restrict__ x, const float* __restrict__ v,
                                                   const int32_t* __restrict__ type, const int32_t* __restrict__ bond,
                                                   float4* __restrict__ X4, float4* __restrict__ W4, int32_t* __restrict__ B)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    X4[i] = make_float4(x[3 * (size_t)i], x[3 * (size_t)i + 1], x[3 * (size_t)i + 2], __int_as_float(type[i]));
    if (W4) {
        float4 w = make_float4(0.f, 0.f, 0.f, __uint_as_float((uint32_t)i));
        if (v) {
            w.x = v[3 * (size_t)i];
            w.y = v[3 * (size_t)i + 1];
            w.z = v[3 * (size_t)i + 2];
        }
        W4[i] = w;
    }
    if (B)
        for (int k = 0; k < max_bonds; ++k) B[(size_t)i * max_bonds + k] = bond[(size_t)i * max_bonds + k];
}

// key = segment * 32 + (local z cell mod 32), segment = tile * S + species; rank = arrival order in that lane list
template <int P>
__global__ void __launch_bounds__(256) ell_key_kernel(MeshParams m, TileParams tp, size_t nsrc, const float4* __restrict__ X4,
                                                      uint32_t* __restrict__ key, uint32_t* __restrict__ rank,
                                                      uint32_t* __restrict__ count)
{
    const size_t s = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= nsrc) return;
    const float4 p = X4[s];
    const int type = __float_as_int(p.w);
    if (type < 0) {
        key[s] = 0xFFFFFFFFu;
        return;
    }
    const float pos[3] = {p.x, p.y, p.z};
    int t[3], rz = 0;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        int cell, b;
        float off;
        index_1d<P>(pos[a], m.inv_h[a], cell, b, off);
        cell = wrap_idx(cell, m.N[a]);
        t[a] = cell / tp.T[a];
        // lane = z of the stencil's first node relative to the tile (the cell for even P, the nearest node for odd P)
        if (a == 2) rz = wrap_idx(b + tp.lo, m.N[2]) - t[2] * tp.T[2];
    }
    const uint32_t tile = (uint32_t)((t[0] * tp.nt[1] + t[1]) * tp.nt[2] + t[2]);
    const uint32_t k = ((tile * (uint32_t)m.S + (uint32_t)type) << 5) | (uint32_t)(rz & 31);
    key[s] = k;
    rank[s] = atomicAdd(&count[k], 1u);
}

// one warp per segment: rounds = min(longest lane list, ceil(fill * mean) + add); out[seg] = 32 * rounds.
// Lanes shorter than `rounds` leave holes; holepref[seg*32 + r] = holes in lanes < r, segholes[seg] = all of them.
// Particles beyond `rounds` in their own lane are placed into those holes by ell_scatter_kernel (they cost a 2-way
// bank conflict in the round they land in, instead of an idle lane slot or a trip through the per-particle kernels).
__global__ void __launch_bounds__(256) ell_rounds_kernel(int nseg, float fill, int add, const uint32_t* __restrict__ count,
                                                         uint32_t* __restrict__ rounds32, uint32_t* __restrict__ holepref,
                                                         uint32_t* __restrict__ segholes, uint32_t* __restrict__ segtick)
{
    const int seg = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (seg >= nseg) return;
    const uint32_t len = count[((size_t)seg << 5) + lane];
    uint32_t mx = len, sum = len;
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, d));
        sum += __shfl_xor_sync(0xffffffffu, sum, d);
    }
    const uint32_t cap = (sum && fill > 0.0f) ? (uint32_t)ceilf(fill * (float)sum * (1.0f / 32.0f)) + (uint32_t)add : 0u;
    const uint32_t rounds = min(mx, cap);
    const uint32_t deficit = rounds > len ? rounds - len : 0u;
    uint32_t incl = deficit;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const uint32_t o = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= d) incl += o;
    }
    holepref[((size_t)seg << 5) + lane] = incl - deficit;
    if (lane == 31) segholes[seg] = incl;
    if (lane == 0) {
        rounds32[seg] = 32u * rounds;
        segtick[seg] = 0u;
    }
    if (seg == 0 && lane == 0) rounds32[nseg] = 0u;
}

// new slot of every source slot: own lane list first, then the holes of the segment, then the overflow tail
__global__ void __launch_bounds__(256) ell_scatter_kernel(size_t nsrc, int nseg, const uint32_t* __restrict__ key,
                                                          const uint32_t* __restrict__ rank, const uint32_t* __restrict__ seg_base,
                                                          const uint32_t* __restrict__ count, const uint32_t* __restrict__ holepref,
                                                          const uint32_t* __restrict__ segholes, uint32_t* __restrict__ segtick,
                                                          const float4* __restrict__ X4src, float4* __restrict__ X4dst,
                                                          uint32_t* __restrict__ inv, uint32_t* __restrict__ totals)
{
    const size_t s = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= nsrc) return;
    const uint32_t k = key[s];
    if (k == 0xFFFFFFFFu) {
        inv[s] = 0xFFFFFFFFu;
        return;
    }
    const uint32_t seg = k >> 5, r = k & 31u, b0 = seg_base[seg], rounds = (seg_base[seg + 1] - b0) >> 5, rk = rank[s];
    uint32_t d;
    if (rk < rounds) {
        d = b0 + rk * 32u + r;
    } else {
        const uint32_t t = atomicAdd(&segtick[seg], 1u);
        if (t < segholes[seg]) {
            const uint32_t* hp = holepref + ((size_t)seg << 5);
            uint32_t lo = 0;   // largest lane with holepref <= t
#pragma unroll
            for (uint32_t step = 16; step > 0; step >>= 1)
                if (hp[lo + step] <= t) lo += step;
            d = b0 + (count[((size_t)seg << 5) + lo] + (t - hp[lo])) * 32u + lo;
        } else {
            d = seg_base[nseg] + atomicAdd(&totals[0], 1u);
        }
    }
    inv[s] = d;
    X4dst[d] = X4src[s];
}

// moves the rest of the state (w + id, bond partner slots remapped through inv) to the new slots
__global__ void __launch_bounds__(256) ell_move_state_kernel(size_t nsrc, int max_bonds, const uint32_t* __restrict__ inv,
                                                             const float4* __restrict__ W4src, const int32_t* __restrict__ Bsrc,
                                                             float4* __restrict__ W4dst, int32_t* __restrict__ Bdst)
{
    const size_t s = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= nsrc) return;
    const uint32_t d = inv[s];
    if (d == 0xFFFFFFFFu) return;
    W4dst[d] = W4src[s];
    for (int k = 0; k < max_bonds; ++k) {
        const int32_t q = Bsrc[s * max_bonds + k];
        Bdst[(size_t)d * max_bonds + k] = q < 0 ? -1 : (int32_t)inv[q];
    }
}

// dst[id[s]][0..2] = src[s].xyz for every occupied slot
__global__ void __launch_bounds__(256) unpermute_kernel(size_t nslots, const float4* __restrict__ W4, const float4* __restrict__ src,
                                                        float* __restrict__ dst)
{
    const size_t s = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= nslots) return;
    const uint32_t id = __float_as_uint(W4[s].w);
    if (id == 0xFFFFFFFFu) return;
    const float4 v = src[s];
    dst[3 * (size_t)id + 0] = v.x;
    dst[3 * (size_t)id + 1] = v.y;
    dst[3 * (size_t)id + 2] = v.z;
}

int exclusive_scan(tild_ctx* c, const uint32_t* in, size_t len, uint32_t* out)
{
    const int nbs = (int)((len + SCAN_CHUNK - 1) / SCAN_CHUNK);
    scan_reduce_kernel<<<nbs, SCAN_THREADS, 0, c->stream>>>(len, in, c->scan_part);
    TILD_LAUNCH_CHECK(c, "scan_reduce_kernel");
    scan_parts_kernel<<<1, 1024, 0, c->stream>>>(nbs, c->scan_part);
    TILD_LAUNCH_CHECK(c, "scan_parts_kernel");
    scan_final_kernel<<<nbs, SCAN_THREADS, 0, c->stream>>>(len, in, c->scan_part, out);
    TILD_LAUNCH_CHECK(c, "scan_final_kernel");
    return TILD_OK;
}

inline unsigned blocks_for(size_t n) { return (unsigned)((n + 255) / 256); }

}  // namespace

int launch_cell_keys(tild_ctx* c, const float* x, uint32_t* key, int32_t* base)
{
    const int n = c->mesh.n;
    if (n == 0) return TILD_OK;
    const int nb = (n + 255) / 256;
    switch (c->mesh.P) {
    case 1: cell_key_kernel<1><<<nb, 256, 0, c->stream>>>(c->mesh, x, key, base); break;
    case 2: cell_key_kernel<2><<<nb, 256, 0, c->stream>>>(c->mesh, x, key, base); break;
    case 3: cell_key_kernel<3><<<nb, 256, 0, c->stream>>>(c->mesh, x, key, base); break;
    default: cell_key_kernel<4><<<nb, 256, 0, c->stream>>>(c->mesh, x, key, base); break;
    }
    TILD_LAUNCH_CHECK(c, "cell_key_kernel");
    return TILD_OK;
}

// Counting sort by cell key: histogram (arrival rank per particle) -> exclusive scan -> scatter.
int launch_counting_sort(tild_ctx* c, const uint32_t* key, size_t nbins, uint32_t* perm, uint32_t* start)
{
    const int n = c->mesh.n;
    const size_t len = nbins + 1;
    TILD_CUDA(c, cudaMemsetAsync(c->count, 0, len * sizeof(uint32_t), c->stream));
    if (n > 0) {
        histogram_kernel<<<(n + 255) / 256, 256, 0, c->stream>>>(n, key, c->count, c->rank);
        TILD_LAUNCH_CHECK(c, "histogram_kernel");
    }
    int rc = exclusive_scan(c, c->count, len, start);
    if (rc) return rc;
    if (n > 0 && perm) {
        scatter_perm_kernel<<<(n + 255) / 256, 256, 0, c->stream>>>(n, key, start, c->rank, perm);
        TILD_LAUNCH_CHECK(c, "scatter_perm_kernel");
    }
    return TILD_OK;
}

int launch_pack(tild_ctx* c, const float* x, const float* v, const int32_t* type, const int32_t* bond, float4* X4, float4* W4,
                int32_t* B)
{
    const int n = c->mesh.n;
    if (n == 0) return TILD_OK;
    pack_kernel<<<(n + 255) / 256, 256, 0, c->stream>>>(n, c->stp.max_bonds, x, v, type, bond, X4, W4, bond ? B : nullptr);
    TILD_LAUNCH_CHECK(c, "pack_kernel");
    return TILD_OK;
}

int launch_build_ell(tild_ctx* c, size_t nsrc, const float4* X4src, float4* X4dst, EllLayout* lay)
{
    const TileParams& tp = c->tile;
    const int nseg = tp.nseg;
    const size_t nbins = (size_t)nseg * 32;
    TILD_CUDA(c, cudaMemsetAsync(c->count, 0, nbins * sizeof(uint32_t), c->stream));
    TILD_CUDA(c, cudaMemsetAsync(c->totals, 0, 4 * sizeof(uint32_t), c->stream));
    if (nsrc > 0) {
        switch (c->mesh.P) {
        case 1: ell_key_kernel<1><<<blocks_for(nsrc), 256, 0, c->stream>>>(c->mesh, tp, nsrc, X4src, c->key, c->rank, c->count); break;
        case 2: ell_key_kernel<2><<<blocks_for(nsrc), 256, 0, c->stream>>>(c->mesh, tp, nsrc, X4src, c->key, c->rank, c->count); break;
        case 3: ell_key_kernel<3><<<blocks_for(nsrc), 256, 0, c->stream>>>(c->mesh, tp, nsrc, X4src, c->key, c->rank, c->count); break;
        default: ell_key_kernel<4><<<blocks_for(nsrc), 256, 0, c->stream>>>(c->mesh, tp, nsrc, X4src, c->key, c->rank, c->count); break;
        }
        TILD_LAUNCH_CHECK(c, "ell_key_kernel");
    }
    uint32_t* rounds32 = c->start;  // [nseg+1] scratch
    ell_rounds_kernel<<<blocks_for((size_t)nseg * 32), 256, 0, c->stream>>>(nseg, tp.enabled ? tp.fill : 0.0f, tp.enabled ? tp.add : 0,
                                                                             c->count, rounds32, c->holepref, c->segholes, c->segtick);
    TILD_LAUNCH_CHECK(c, "ell_rounds_kernel");
    int rc = exclusive_scan(c, rounds32, (size_t)nseg + 1, lay->seg_base);
    if (rc) return rc;
    // holes of the ELL region: type = -1 (all-ones bit pattern); the tail is written densely
    TILD_CUDA(c, cudaMemsetAsync(X4dst, 0xFF, tp.cap_ell * sizeof(float4), c->stream));
    if (nsrc > 0) {
        ell_scatter_kernel<<<blocks_for(nsrc), 256, 0, c->stream>>>(nsrc, nseg, c->key, c->rank, lay->seg_base, c->count, c->holepref,
                                                                    c->segholes, c->segtick, X4src, X4dst, c->inv, c->totals);
        TILD_LAUNCH_CHECK(c, "ell_scatter_kernel");
    }
    uint32_t h[2] = {0, 0};
    TILD_CUDA(c, cudaMemcpyAsync(&h[0], lay->seg_base + nseg, sizeof(uint32_t), cudaMemcpyDeviceToHost, c->stream));
    TILD_CUDA(c, cudaMemcpyAsync(&h[1], c->totals, sizeof(uint32_t), cudaMemcpyDeviceToHost, c->stream));
    TILD_CUDA(c, cudaStreamSynchronize(c->stream));
    lay->total_ell = h[0];
    lay->n_ovf = h[1];
    if (lay->total_ell > tp.cap_ell || lay->used() > tp.cap)
        return tild_fail(c, TILD_ENOMEM, "slab layout needs %zu + %zu slots, capacity %zu + %zu", lay->total_ell, lay->n_ovf,
                         tp.cap_ell, tp.cap - tp.cap_ell);
    return TILD_OK;
}

int launch_reorder(tild_ctx* c)
{
    const int a = c->cur, b = 1 - c->cur;
    const size_t nsrc = c->lay.used();
    int rc = launch_build_ell(c, nsrc, c->X4[a], c->X4[b], &c->lay);
    if (rc) return rc;
    c->steps_since_sort = 0;
    const TileParams& tp = c->tile;
    TILD_CUDA(c, cudaMemsetAsync(c->W4[b], 0xFF, tp.cap_ell * sizeof(float4), c->stream));
    if (nsrc > 0) {
        ell_move_state_kernel<<<blocks_for(nsrc), 256, 0, c->stream>>>(nsrc, c->stp.max_bonds, c->inv, c->W4[a], c->B[a], c->W4[b],
                                                                       c->B[b]);
        TILD_LAUNCH_CHECK(c, "ell_move_state_kernel");
    }
    // the fused step never writes holes, so the other buffer pair must carry the hole markers too
    TILD_CUDA(c, cudaMemsetAsync(c->X4[a], 0xFF, tp.cap_ell * sizeof(float4), c->stream));
    TILD_CUDA(c, cudaMemsetAsync(c->W4[a], 0xFF, tp.cap_ell * sizeof(float4), c->stream));
    c->cur = b;
    return TILD_OK;
}

int launch_unpermute(tild_ctx* c, const float4* src, float* dst)
{
    const size_t ns = c->lay.used();
    if (ns == 0) return TILD_OK;
    unpermute_kernel<<<blocks_for(ns), 256, 0, c->stream>>>(ns, c->W4[c->cur], src, dst);
    TILD_LAUNCH_CHECK(c, "unpermute_kernel");
    return TILD_OK;
}

size_t tild_scan_scratch_entries(size_t nbins)
{
    const size_t len = nbins + 1;
    return (len + SCAN_CHUNK - 1) / SCAN_CHUNK + 16;
}
