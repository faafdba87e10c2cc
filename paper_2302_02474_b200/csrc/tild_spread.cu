// a2: particle -> mesh spread.  PAPER.md L223: "at each time-step, every particle assigns
// its density contribution to nearby grid points, using a spline interpolation scheme"; Eq. 1 L110.
// grid[J][g] = sum_{i in J} W_x W_y W_z  (raw weights), g = (ix*Ny + iy)*Nz + iz.
#include "tild_internal.cuh"

namespace {

// Baseline: one thread per particle, P^3 global reductions (REDG.E.ADD.F32 resolves in L2).  With the
// particle arrays kept in cell order by launch_reorder, neighbouring threads hit neighbouring lines.
template <int P>
__global__ void __launch_bounds__(256) spread_naive_kernel(MeshParams m, const float* __restrict__ x,
                                                           const int32_t* __restrict__ type, float* __restrict__ grid)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= m.n) return;
    int cell, b[3];
    float t, w[3][P];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        index_1d<P>(x[3 * (size_t)i + a], m.inv_h[a], cell, b[a], t);
        weights_1d<P>(t, w[a]);
    }
    float* g = grid + (size_t)type[i] * m.M;
    int iz[P];
#pragma unroll
    for (int j = 0; j < P; ++j) iz[j] = wrap_idx(b[2] + j, m.N[2]);
#pragma unroll
    for (int jx = 0; jx < P; ++jx) {
        const size_t ox = (size_t)wrap_idx(b[0] + jx, m.N[0]) * m.N[1];
#pragma unroll
        for (int jy = 0; jy < P; ++jy) {
            const size_t row = (ox + wrap_idx(b[1] + jy, m.N[1])) * m.N[2];
            const float wxy = w[0][jx] * w[1][jy];
#pragma unroll
            for (int jz = 0; jz < P; ++jz) atomicAdd(g + row + iz[jz], wxy * w[2][jz]);
        }
    }
}

}  // namespace

int launch_spread(tild_ctx* c, const float* x, const int32_t* type, float* grid)
{
    const int n = c->mesh.n;
    TILD_CUDA(c, cudaMemsetAsync(grid, 0, sizeof(float) * c->M * c->mesh.S, c->stream));
    if (n == 0) return TILD_OK;
    const int nb = (n + 255) / 256;
    switch (c->mesh.P) {
    case 1: spread_naive_kernel<1><<<nb, 256, 0, c->stream>>>(c->mesh, x, type, grid); break;
    case 2: spread_naive_kernel<2><<<nb, 256, 0, c->stream>>>(c->mesh, x, type, grid); break;
    case 3: spread_naive_kernel<3><<<nb, 256, 0, c->stream>>>(c->mesh, x, type, grid); break;
    default: spread_naive_kernel<4><<<nb, 256, 0, c->stream>>>(c->mesh, x, type, grid); break;
    }
    TILD_LAUNCH_CHECK(c, "spread_naive_kernel");
    return TILD_OK;
}
