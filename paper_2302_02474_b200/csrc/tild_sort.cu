// a1: canonical fp32 index map, cell keys, counting sort by cell (the stage call tild_index_map),
// and the segment (tile, species) ordering of the internal particle state that the tile kernels run on.
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

// caller arrays -> slots [0, n): slot i holds particle id i.  A type outside [0, S) or a partner outside [-1, n) is
// replaced by 0 / -1 (so that no later kernel indexes out of bounds) and reported through *bad.
__global__ void __launch_bounds__(256) pack_kernel(int n, int S, int max_bonds, const float* __restrict__ x, const float* __restrict__ v,
                                                   const int32_t* __restrict__ type, const int32_t* __restrict__ bond,
                                                   float4* __restrict__ X4, float4* __restrict__ W4, int32_t* __restrict__ B,
                                                   uint32_t* __restrict__ bad)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int32_t ty = type[i];
    bool wrong = ty < 0 || ty >= S;
    if (wrong) ty = 0;
    X4[i] = make_float4(x[3 * (size_t)i], x[3 * (size_t)i + 1], x[3 * (size_t)i + 2], __int_as_float(ty));
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
        for (int k = 0; k < max_bonds; ++k) {
            int32_t q = bond[(size_t)i * max_bonds + k];
            if (q < -1 || q >= n) {
                wrong = true;
                q = -1;
            }
            B[(size_t)i * max_bonds + k] = q;
        }
    if (wrong) atomicOr(bad, 1u);
}

// key = segment = tile * S + species; rank = arrival order in the segment (one atomic per distinct key per warp)
template <int P>
__global__ void __launch_bounds__(256) seg_key_kernel(MeshParams m, TileParams tp, const float4* __restrict__ X4,
                                                      uint32_t* __restrict__ key, uint32_t* __restrict__ rank,
                                                      uint32_t* __restrict__ count)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    uint32_t k = 0xFFFFFFFFu;
    if (s < m.n) {
        const float4 p = X4[s];
        const float pos[3] = {p.x, p.y, p.z};
        int t[3];
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            int cell, b;
            float off;
            index_1d<P>(pos[a], m.inv_h[a], cell, b, off);
            t[a] = wrap_idx(cell, m.N[a]) / tp.T[a];
        }
        k = (uint32_t)((t[0] * tp.nt[1] + t[1]) * tp.nt[2] + t[2]) * (uint32_t)m.S + (uint32_t)__float_as_int(p.w);
    }
    const unsigned peers = __match_any_sync(0xffffffffu, k);
    const int lane = threadIdx.x & 31, leader = __ffs(peers) - 1;
    uint32_t base = 0;
    if (lane == leader && k != 0xFFFFFFFFu) base = atomicAdd(&count[k], (uint32_t)__popc(peers));
    base = __shfl_sync(0xffffffffu, base, leader);
    if (s < m.n) {
        key[s] = k;
        rank[s] = base + (uint32_t)__popc(peers & ((1u << lane) - 1u));
    }
}

__global__ void __launch_bounds__(256) seg_scatter_kernel(int n, const uint32_t* __restrict__ key, const uint32_t* __restrict__ rank,
                                                          const uint32_t* __restrict__ seg_base, const float4* __restrict__ X4src,
                                                          float4* __restrict__ X4dst, uint32_t* __restrict__ inv)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    const uint32_t d = seg_base[key[s]] + rank[s];
    inv[s] = d;
    X4dst[d] = X4src[s];
}

// ---- order-preserving re-sort --------------------------------------------------------------------------------------
// The re-sort of the timed path keeps the particles that stay in their segment ("stayers": nearly all of them, the state
// was sorted a few steps ago) in the order they had, and appends the ones that changed segment behind them.  With ranks
// handed out by atomics in arrival order every re-sort cut the order into warp-sized pieces and shuffled those, and the
// bond partners of the fused step -- chain neighbours, adjacent in memory after the first sort -- drifted apart: the
// interpolation stage of C4 went from 0.549 to 0.606 ms over 300 steps.  A stayer's rank is the number of stayers in front
// of it in its (old = new) segment.
// One CTA per OLD segment g walks its slots in order: a stayer's rank is the running count of stayers in front of it.
__global__ void __launch_bounds__(256) seg_key_stable_kernel(MeshParams m, TileParams tp, const float4* __restrict__ X4,
                                                             const uint32_t* __restrict__ old_base, uint32_t* __restrict__ key,
                                                             uint32_t* __restrict__ rank, uint32_t* __restrict__ count,
                                                             uint32_t* __restrict__ count_m, uint32_t* __restrict__ stayers)
{
    __shared__ uint32_t wsum[8];
    const uint32_t g = blockIdx.x, lo = old_base[g], hi = old_base[g + 1];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    uint32_t running = 0;                                          // uniform
    for (uint32_t c0 = lo; c0 < hi; c0 += 256) {
        const uint32_t s = c0 + threadIdx.x;
        uint32_t k = 0xFFFFFFFFu;
        if (s < hi) {
            const float4 p = X4[s];
            const float pos[3] = {p.x, p.y, p.z};
            int t[3];
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                int cell, b;
                float off;
                index_1d<4>(pos[a], m.inv_h[a], cell, b, off);   // the cell does not depend on the order P
                t[a] = wrap_idx(cell, m.N[a]) / tp.T[a];
            }
            k = (uint32_t)((t[0] * tp.nt[1] + t[1]) * tp.nt[2] + t[2]) * (uint32_t)m.S + (uint32_t)__float_as_int(p.w);
        }
        const bool stayer = k == g;
        const unsigned bal = __ballot_sync(0xffffffffu, stayer);
        if (lane == 0) wsum[wid] = (uint32_t)__popc(bal);
        __syncthreads();
        uint32_t before = 0, total = 0;
#pragma unroll
        for (int w = 0; w < 8; ++w) {
            const uint32_t v = wsum[w];
            before += w < wid ? v : 0u;
            total += v;
        }
        __syncthreads();
        if (s < hi) {
            key[s] = k;
            if (stayer) {
                rank[s] = running + before + (uint32_t)__popc(bal & ((1u << lane) - 1u));
            } else {                                               // moved in from another segment: behind the stayers, arrival order
                atomicAdd(&count[k], 1u);
                rank[s] = 0x80000000u | atomicAdd(&count_m[k], 1u);
            }
        }
        running += total;
    }
    if (threadIdx.x == 0) {
        stayers[g] = running;
        if (running) atomicAdd(&count[g], running);
    }
}

__global__ void __launch_bounds__(256) seg_scatter_stable_kernel(int n, const uint32_t* __restrict__ key, const uint32_t* __restrict__ rank,
                                                                 const uint32_t* __restrict__ stayers, const uint32_t* __restrict__ seg_base,
                                                                 const float4* __restrict__ X4src, float4* __restrict__ X4dst,
                                                                 uint32_t* __restrict__ inv)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    const uint32_t k = key[s], r = rank[s];
    const uint32_t d = seg_base[k] + ((r & 0x80000000u) ? stayers[k] + (r & 0x7FFFFFFFu) : r);
    inv[s] = d;
    X4dst[d] = X4src[s];
}

// moves the rest of the state (w + id, bond partner slots remapped through inv) to the new slots
__global__ void __launch_bounds__(256) move_state_kernel(int n, int max_bonds, const uint32_t* __restrict__ inv,
                                                         const float4* __restrict__ W4src, const int32_t* __restrict__ Bsrc,
                                                         float4* __restrict__ W4dst, int32_t* __restrict__ Bdst)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    const uint32_t d = inv[s];
    W4dst[d] = W4src[s];
    for (int k = 0; k < max_bonds; ++k) {
        const int32_t q = Bsrc[(size_t)s * max_bonds + k];
        Bdst[(size_t)d * max_bonds + k] = q < 0 ? -1 : (int32_t)inv[q];
    }
}

// dst[id[s]][0..2] = src[s].xyz
__global__ void __launch_bounds__(256) unpermute_kernel(int n, const float4* __restrict__ W4, const float4* __restrict__ src,
                                                        float* __restrict__ dst)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    const uint32_t id = __float_as_uint(W4[s].w);
    const float4 v = src[s];
    dst[3 * (size_t)id + 0] = v.x;
    dst[3 * (size_t)id + 1] = v.y;
    dst[3 * (size_t)id + 2] = v.z;
}

// id[s] = original particle id held by slot s
__global__ void __launch_bounds__(256) slot_ids_kernel(int n, const float4* __restrict__ W4, uint32_t* __restrict__ id)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s < n) id[s] = __float_as_uint(W4[s].w);
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
    case 4: cell_key_kernel<4><<<nb, 256, 0, c->stream>>>(c->mesh, x, key, base); break;
    default: cell_key_kernel<5><<<nb, 256, 0, c->stream>>>(c->mesh, x, key, base); break;
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
    pack_kernel<<<(n + 255) / 256, 256, 0, c->stream>>>(n, c->mesh.S, c->stp.max_bonds, x, v, type, bond, X4, W4, bond ? B : nullptr,
                                                          c->drift_count + 2);
    TILD_LAUNCH_CHECK(c, "pack_kernel");
    return TILD_OK;
}

int launch_segment_sort(tild_ctx* c, const float4* X4src, float4* X4dst, SegLayout* lay)
{
    const TileParams& tp = c->tile;
    const int n = c->mesh.n, nseg = tp.nseg;
    TILD_CUDA(c, cudaMemsetAsync(c->count, 0, ((size_t)nseg + 1) * sizeof(uint32_t), c->stream));
    if (n > 0) {
        switch (c->mesh.P) {
        case 1: seg_key_kernel<1><<<blocks_for(n), 256, 0, c->stream>>>(c->mesh, tp, X4src, c->key, c->rank, c->count); break;
        case 2: seg_key_kernel<2><<<blocks_for(n), 256, 0, c->stream>>>(c->mesh, tp, X4src, c->key, c->rank, c->count); break;
        case 3: seg_key_kernel<3><<<blocks_for(n), 256, 0, c->stream>>>(c->mesh, tp, X4src, c->key, c->rank, c->count); break;
        case 4: seg_key_kernel<4><<<blocks_for(n), 256, 0, c->stream>>>(c->mesh, tp, X4src, c->key, c->rank, c->count); break;
        default: seg_key_kernel<5><<<blocks_for(n), 256, 0, c->stream>>>(c->mesh, tp, X4src, c->key, c->rank, c->count); break;
        }
        TILD_LAUNCH_CHECK(c, "seg_key_kernel");
    }
    int rc = exclusive_scan(c, c->count, (size_t)nseg + 1, lay->seg_base);
    if (rc) return rc;
    if (n > 0) {
        seg_scatter_kernel<<<blocks_for(n), 256, 0, c->stream>>>(n, c->key, c->rank, lay->seg_base, X4src, X4dst, c->inv);
        TILD_LAUNCH_CHECK(c, "seg_scatter_kernel");
    }
    return TILD_OK;
}

// re-sort of a state that c->lay describes (sorted at the last re-sort): stayers keep their order
int launch_segment_resort(tild_ctx* c, const float4* X4src, float4* X4dst, SegLayout* lay)
{
    const TileParams& tp = c->tile;
    const int n = c->mesh.n, nseg = tp.nseg;
    if (n == 0) return launch_segment_sort(c, X4src, X4dst, lay);
    uint32_t* old_base = c->start;                               // [nseg + 1] | stayers [nseg]
    uint32_t* stayers = c->start + (size_t)nseg + 2;
    uint32_t* count_m = c->count + (size_t)nseg + 2;             // count [nseg + 1] | count_m [nseg]
    TILD_CUDA(c, cudaMemcpyAsync(old_base, lay->seg_base, ((size_t)nseg + 1) * sizeof(uint32_t), cudaMemcpyDeviceToDevice, c->stream));
    TILD_CUDA(c, cudaMemsetAsync(c->count, 0, (2 * (size_t)nseg + 4) * sizeof(uint32_t), c->stream));
    seg_key_stable_kernel<<<nseg, 256, 0, c->stream>>>(c->mesh, tp, X4src, old_base, c->key, c->rank, c->count, count_m, stayers);
    TILD_LAUNCH_CHECK(c, "seg_key_stable_kernel");
    int rc = exclusive_scan(c, c->count, (size_t)nseg + 1, lay->seg_base);
    if (rc) return rc;
    seg_scatter_stable_kernel<<<blocks_for(n), 256, 0, c->stream>>>(n, c->key, c->rank, stayers, lay->seg_base, X4src, X4dst, c->inv);
    TILD_LAUNCH_CHECK(c, "seg_scatter_stable_kernel");
    return TILD_OK;
}

int launch_reorder(tild_ctx* c)
{
    const int a = c->cur, b = 1 - c->cur, n = c->mesh.n;
    int rc = (c->lay_valid && !(c->prm.flags & TILD_FLAG_ARRIVAL_SORT)) ? launch_segment_resort(c, c->X4[a], c->X4[b], &c->lay)
                                                                        : launch_segment_sort(c, c->X4[a], c->X4[b], &c->lay);
    c->lay_valid = true;
    if (rc) return rc;
    c->steps_since_sort = 0;
    c->resorts_since_defrag++;
    if (n > 0) {
        move_state_kernel<<<blocks_for(n), 256, 0, c->stream>>>(n, c->stp.max_bonds, c->inv, c->W4[a], c->B[a], c->W4[b], c->B[b]);
        TILD_LAUNCH_CHECK(c, "move_state_kernel");
    }
    c->cur = b;
    return launch_slot_of_id(c);   // id -> slot map of the extra mesh interactions (no-op without TILD_FLAG_EXTRAS)
}

// slot s -> slot id(s): the state in the order tild_set_state packs it (particle id = slot)
__global__ void __launch_bounds__(256) to_id_order_kernel(int n, int max_bonds, const float4* __restrict__ X4src, const float4* __restrict__ W4src,
                                                          const int32_t* __restrict__ Bsrc, float4* __restrict__ X4dst,
                                                          float4* __restrict__ W4dst, int32_t* __restrict__ Bdst)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    const float4 w = W4src[s];
    const uint32_t id = __float_as_uint(w.w);
    X4dst[id] = X4src[s];
    W4dst[id] = w;
    for (int k = 0; k < max_bonds; ++k) {
        const int32_t q = Bsrc[(size_t)s * max_bonds + k];
        Bdst[(size_t)id * max_bonds + k] = q < 0 ? -1 : (int32_t)__float_as_uint(W4src[q].w);
    }
}

// Every TILD_DEFRAG_EVERY re-sorts the state is put back into particle-id order and sorted from there, as tild_set_state
// does: the order-preserving re-sorts keep chain neighbours together only until they cross a tile boundary (they come back
// to the end of their segment), and this restores the order of a fresh state (C4: interp 0.577 -> 0.543 ms after 300 steps).
// Leaves cur where it was (two buffer flips).
int launch_defrag(tild_ctx* c)
{
    const int a = c->cur, b = 1 - c->cur, n = c->mesh.n;
    if (n > 0) {
        to_id_order_kernel<<<blocks_for(n), 256, 0, c->stream>>>(n, c->stp.max_bonds, c->X4[a], c->W4[a], c->B[a], c->X4[b], c->W4[b], c->B[b]);
        TILD_LAUNCH_CHECK(c, "to_id_order_kernel");
    }
    c->cur = b;
    c->lay_valid = false;
    const int rc = launch_reorder(c);
    c->resorts_since_defrag = 0;
    return rc;
}

int launch_unpermute(tild_ctx* c, const float4* src, float* dst)
{
    const int n = c->mesh.n;
    if (n == 0) return TILD_OK;
    unpermute_kernel<<<blocks_for(n), 256, 0, c->stream>>>(n, c->W4[c->cur], src, dst);
    TILD_LAUNCH_CHECK(c, "unpermute_kernel");
    return TILD_OK;
}

int launch_slot_ids(tild_ctx* c, uint32_t* id)
{
    const int n = c->mesh.n;
    if (n == 0) return TILD_OK;
    slot_ids_kernel<<<blocks_for(n), 256, 0, c->stream>>>(n, c->W4[c->cur], id);
    TILD_LAUNCH_CHECK(c, "slot_ids_kernel");
    return TILD_OK;
}

size_t tild_scan_scratch_entries(size_t nbins)
{
    const size_t len = nbins + 1;
    return (len + SCAN_CHUNK - 1) / SCAN_CHUNK + 16;
}
