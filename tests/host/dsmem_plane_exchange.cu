// Measurement behind the 3-pass ("T1") decision of DESIGN.md section 9: the data movement a fused
// y-fwd . z . multiply . z-inv . y-inv kernel would need at C3 (256x256x64 fp32), WITHOUT the transforms.
//
// One thread-block cluster of 8 CTAs holds one pair plane after the y transform: Ny x nz x 3 quads = 512 x 64 x 3 x 16 B
// = 1.5 MB, CTA j owning the lines of z in [8j, 8j+8) as P[py][c*8 + z_local] (196,608 B).  The z stage needs whole z columns:
// CTA r gathers, for its 64 columns py in groups of TY = 4, the 8 z-slices from the 8 CTAs of the cluster (7 of them
// through distributed shared memory) into a work tile W[z][c*TY + ty] (24,576 B), "transforms" it (here: x -> -x, so that
// the round trip can be checked), and scatters it back.  Two cluster barriers per plane stand for the y-phase / z-phase
// boundaries.  Prints the time per plane and the DSMEM bytes per clock per SM it corresponds to.
//
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o dsmem_plane_exchange dsmem_plane_exchange.cu && ./dsmem_plane_exchange
#include <cooperative_groups.h>
#include <cuda_runtime.h>
#include <cstdio>
#include <vector>
namespace cg = cooperative_groups;

constexpr int NY = 512, NZ = 64, CL = 8, ZL = NZ / CL, LINES = 3 * ZL, TY = 4, NT = 256;
constexpr int PLANE_Q = NY * LINES;              // quads of the plane share of one CTA
constexpr int WORK_Q = NZ * 3 * TY;              // quads of the z work tile

__global__ void __launch_bounds__(NT) k_exchange(float4* out, int planes)
{
    extern __shared__ float4 smem[];
    float4* P = smem;                            // [py][line]
    float4* W = smem + PLANE_Q;                  // [z][c * TY + ty]
    cg::cluster_group cluster = cg::this_cluster();
    const int r = (int)cluster.block_rank(), tid = threadIdx.x;
    const int cid = blockIdx.x / CL;
    for (int i = tid; i < PLANE_Q; i += NT) { const float v = (float)(i + r * PLANE_Q); P[i] = make_float4(v, v + 0.25f, -v, 1.0f + cid); }
    cluster.sync();
    for (int it = 0; it < planes; ++it) {
        for (int g = 0; g < NY / CL / TY; ++g) {                   // 16 column groups of this CTA
            const int py0 = r * (NY / CL) + g * TY;
            // gather: W[z][c*TY+ty] = P_j[py0+ty][c*ZL + zl],  z = j*ZL + zl
            for (int i = tid; i < WORK_Q; i += NT) {
                const int line = i % LINES, rest = i / LINES, ty = rest % TY, j = rest / TY;
                const int c = line / ZL, zl = line % ZL;
                const float4* src = cluster.map_shared_rank(P, j);
                W[(j * ZL + zl) * (3 * TY) + c * TY + ty] = src[(py0 + ty) * LINES + line];
            }
            __syncthreads();
            for (int i = tid; i < WORK_Q; i += NT) { float4 v = W[i]; v.x = -v.x; v.y = -v.y; v.z = -v.z; W[i] = v; }   // the z stage's stand-in
            __syncthreads();
            for (int i = tid; i < WORK_Q; i += NT) {
                const int line = i % LINES, rest = i / LINES, ty = rest % TY, j = rest / TY;
                const int c = line / ZL, zl = line % ZL;
                float4* dst = cluster.map_shared_rank(P, j);
                dst[(py0 + ty) * LINES + line] = W[(j * ZL + zl) * (3 * TY) + c * TY + ty];
            }
            __syncthreads();
        }
        cluster.sync();                                            // z phase done: every CTA's plane share is complete again
        cluster.sync();                                            // (y inverse . next plane's y forward would run here)
    }
    if (out) for (int i = tid; i < PLANE_Q; i += NT) out[(size_t)blockIdx.x * PLANE_Q + i] = P[i];
}

int main()
{
    int dev = 0, sms = 0, khz = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, dev);
    const int smem = (PLANE_Q + WORK_Q) * (int)sizeof(float4);
    if (cudaFuncSetAttribute(k_exchange, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess) { printf("FAIL smem %d\n", smem); return 1; }
    cudaLaunchConfig_t cfg = {};
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension; at[0].val.clusterDim.x = CL; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1; cfg.blockDim = dim3(NT); cfg.dynamicSmemBytes = smem;
    int nclusters = 0;
    cfg.gridDim = dim3(CL * (sms / CL));
    if (cudaOccupancyMaxActiveClusters(&nclusters, k_exchange, &cfg) != cudaSuccess || nclusters < 1) { printf("FAIL no cluster of %d CTAs with %d bytes fits\n", CL, smem); return 1; }
    cfg.gridDim = dim3(CL * nclusters);
    float4* out = nullptr;
    cudaMalloc(&out, (size_t)CL * nclusters * PLANE_Q * sizeof(float4));
    // correctness: an odd number of planes negates x, y, z of every element once per plane -> sign (-1)^planes
    float4* none = nullptr; int one = 3;
    cudaLaunchKernelEx(&cfg, k_exchange, out, one);
    if (cudaDeviceSynchronize() != cudaSuccess) { printf("FAIL launch: %s\n", cudaGetErrorString(cudaGetLastError())); return 1; }
    std::vector<float4> h((size_t)CL * nclusters * PLANE_Q);
    cudaMemcpy(h.data(), out, h.size() * sizeof(float4), cudaMemcpyDeviceToHost);
    for (size_t b = 0; b < (size_t)CL * nclusters; ++b)
        for (int i = 0; i < PLANE_Q; i += 97) {
            const float v = (float)(i + (int)(b % CL) * PLANE_Q);
            const float4 q = h[b * PLANE_Q + i];
            if (q.x != -v || q.y != -(v + 0.25f) || q.z != v || q.w != 1.0f + (float)(b / CL)) { printf("FAIL data at block %zu quad %d\n", b, i); return 1; }
        }
    cudaEvent_t a, b; cudaEventCreate(&a); cudaEventCreate(&b);
    const int planes = 64;
    cudaLaunchKernelEx(&cfg, k_exchange, none, 4);
    cudaEventRecord(a);
    cudaLaunchKernelEx(&cfg, k_exchange, none, planes);
    cudaEventRecord(b); cudaDeviceSynchronize();
    float ms = 0; cudaEventElapsedTime(&ms, a, b);
    const double us_plane = ms * 1e3 / planes;
    const double remote_bytes = 2.0 * (CL - 1) / CL * PLANE_Q * sizeof(float4);      // per CTA per plane, read + written remotely
    printf("OK clusters %d of %d CTAs (%d SMs), smem %d B per CTA; %.2f us per pair plane per cluster; DSMEM %.1f B/clk/SM at %.0f MHz; "
           "C3 (129 pair planes): %.1f us per apply for the exchange alone\n",
           nclusters, CL, sms, smem, us_plane, remote_bytes / (us_plane * 1e-6 * khz * 1e3), khz / 1e3, us_plane * ((129 + nclusters - 1) / nclusters));
    return 0;
}
