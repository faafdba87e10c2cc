// Stand-alone probe, not part of libtild.so (profiles/r2_variants.md, "Interleaved float4 image"): shared-memory pipe time of
// one P = 4 stencil gather per lane for (A) three component planes read with scalar LDS on rotation-group banks -- what
// interp_rot_kernel does -- and (B) an interleaved (fx, fy, fz, pad) float4 image read with LDS.128.
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -std=c++17 -o /tmp/probe_lds paper_2302_02474_b200/csrc/probe_lds.cu && /tmp/probe_lds
#include <cstdio>
#include <cuda_runtime.h>
constexpr int EX = 11, EY = 19, EZ = 40, CS = EX * EY * EZ;
// A: three component planes, scalar LDS, lanes on distinct banks (rotation-group placement)
__global__ void __launch_bounds__(256, 2) probeA(float* out, int iters)
{
    extern __shared__ float s[];
    for (int i = threadIdx.x; i < 3 * CS; i += 256) s[i] = (float)(i & 7);
    __syncthreads();
    const int lane = threadIdx.x & 31;
    float a0 = 0, a1 = 0, a2 = 0;
    int off = ((lane & 7) + 8 * 0) + ((lane >> 3) * 0);   // bank = lane&7 + 8*(lane>>3) via row rotation below
    for (int it = 0; it < iters; ++it) {
        const int base = ((it * 7) % 6) * EY * EZ + ((it * 5) % 14) * EZ + (lane & 7) + 8 * ((it * 3) & 3);
#pragma unroll
        for (int jx = 0; jx < 4; ++jx)
#pragma unroll
            for (int jy = 0; jy < 4; ++jy) {
                const float* f = s + base + jx * EY * EZ + ((jy + (lane >> 3)) & 3) * EZ;
                const float w = (float)(jx + jy);
#pragma unroll
                for (int jz = 0; jz < 4; ++jz) {
                    a0 = fmaf(f[jz], w, a0);
                    a1 = fmaf(f[CS + jz], w, a1);
                    a2 = fmaf(f[2 * CS + jz], w, a2);
                }
            }
    }
    out[blockIdx.x * 256 + threadIdx.x] = a0 + a1 + a2 + off;
}
// B: interleaved float4 (fx, fy, fz, pad) image (8 x 8 x 32 tile + halo = 11 x 11 x 36 nodes so that it fits), LDS.128
__global__ void __launch_bounds__(256, 2) probeB(float* out, int iters)
{
    extern __shared__ float4 s4[];
    constexpr int BY = 11, BZ = 36, N4 = 11 * BY * BZ;
    for (int i = threadIdx.x; i < N4; i += 256) s4[i] = make_float4(1.f, 2.f, 3.f, 0.f);
    __syncthreads();
    const int lane = threadIdx.x & 31;
    float a0 = 0, a1 = 0, a2 = 0;
    for (int it = 0; it < iters; ++it) {
        // quarter-warp lanes on distinct 16-byte bank groups: node index mod 8 = lane & 7
        const int base = ((it * 7) % 6) * BY * BZ + ((it * 5) % 6) * BZ + (lane & 7) + 8 * ((it * 3) & 3);
#pragma unroll
        for (int jx = 0; jx < 4; ++jx)
#pragma unroll
            for (int jy = 0; jy < 4; ++jy) {
                const float4* f = s4 + base + jx * BY * BZ + jy * BZ;
                const float w = (float)(jx + jy);
#pragma unroll
                for (int jz = 0; jz < 4; ++jz) {
                    const float4 v = f[jz];
                    a0 = fmaf(v.x, w, a0);
                    a1 = fmaf(v.y, w, a1);
                    a2 = fmaf(v.z, w, a2);
                }
            }
    }
    out[blockIdx.x * 256 + threadIdx.x] = a0 + a1 + a2;
}
int main()
{
    float* out;
    cudaMalloc(&out, 296 * 256 * 4);
    const int iters = 2000;
    const size_t smA = 3 * CS * 4, smB = 11 * 11 * 36 * 16;
    cudaFuncSetAttribute(probeA, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smA);
    cudaFuncSetAttribute(probeB, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smB);
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    for (int rep = 0; rep < 2; ++rep) {
        float ms;
        cudaEventRecord(e0); probeA<<<296, 256, smA>>>(out, iters); cudaEventRecord(e1); cudaEventSynchronize(e1);
        cudaEventElapsedTime(&ms, e0, e1);
        // per SM: 2 CTAs x 8 warps x iters warp-gathers
        printf("A 3 planes LDS.32 : %.3f ms, %.1f clk per warp-gather per SM (1965 MHz)  smem %zu\n", ms, ms * 1e-3 * 1.965e9 / (16.0 * iters), smA);
        cudaEventRecord(e0); probeB<<<296, 256, smB>>>(out, iters); cudaEventRecord(e1); cudaEventSynchronize(e1);
        cudaEventElapsedTime(&ms, e0, e1);
        printf("B float4   LDS.128: %.3f ms, %.1f clk per warp-gather per SM  smem %zu  err %s\n", ms, ms * 1e-3 * 1.965e9 / (16.0 * iters), smB, cudaGetErrorString(cudaGetLastError()));
    }
    return 0;
}
