// exchange_bench.cu — micro-benchmark behind DESIGN.md 6 "Why no warp-shuffle butterflies": the 16 x 16 exchange between the
// two factors of a pencil DFT (16 lanes x 16 complex values each), done (a) through shared memory as the pass kernels do
// (one STS.64 + one LDS.64 per element, conflict-free pitch) and (b) by a four-stage warp-shuffle butterfly transpose
// (4 SHFL.32 + 2 selects per element).  Prints one JSON line with the time per element of both and checks that both
// produce the transpose.  Stand-alone: nvcc -O3 -gencode arch=compute_100a,code=sm_100a exchange_bench.cu -o exchange_bench
#include <cuda_runtime.h>

#include <cstdio>
#include <vector>

constexpr int kIters = 256;
constexpr int kThreads = 256;

__device__ __forceinline__ void init(float2 (&v)[16], int gid) {
#pragma unroll
    for (int j = 0; j < 16; ++j) v[j] = make_float2((float)(gid * 16 + j), (float)(-(gid * 16 + j)));
}

// (a) through shared memory: lane r of a 16-lane group writes row r, reads column r
__global__ void __launch_bounds__(kThreads) k_smem(float2* out, int iters) {
    __shared__ float2 tile[kThreads / 16][16 * 17];
    const int lane16 = threadIdx.x & 15, grp = threadIdx.x >> 4;
    float2 v[16];
    init(v, blockIdx.x * kThreads + threadIdx.x);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int j = 0; j < 16; ++j) tile[grp][lane16 * 17 + j] = v[j];
        __syncwarp();
#pragma unroll
        for (int j = 0; j < 16; ++j) v[j] = tile[grp][j * 17 + lane16];
        __syncwarp();
    }
    float2* o = out + (size_t)(blockIdx.x * kThreads + threadIdx.x) * 16;
#pragma unroll
    for (int j = 0; j < 16; ++j) o[j] = v[j];
}

// (b) warp shuffles: butterfly transpose, stages d = 8, 4, 2, 1
template <int D>
__device__ __forceinline__ void stage(float2 (&v)[16], int lane16) {
    const bool up = (lane16 & D) != 0;
#pragma unroll
    for (int j = 0; j < 16; ++j) {
        if ((j & D) != 0) continue;
        const float2 send = up ? v[j] : v[j + D];
        float2 recv;
        recv.x = __shfl_xor_sync(0xffffffffu, send.x, D);
        recv.y = __shfl_xor_sync(0xffffffffu, send.y, D);
        if (up) v[j] = recv; else v[j + D] = recv;
    }
}
__global__ void __launch_bounds__(kThreads) k_shfl(float2* out, int iters) {
    const int lane16 = threadIdx.x & 15;
    float2 v[16];
    init(v, blockIdx.x * kThreads + threadIdx.x);
    for (int it = 0; it < iters; ++it) {
        stage<8>(v, lane16); stage<4>(v, lane16); stage<2>(v, lane16); stage<1>(v, lane16);
    }
    float2* o = out + (size_t)(blockIdx.x * kThreads + threadIdx.x) * 16;
#pragma unroll
    for (int j = 0; j < 16; ++j) o[j] = v[j];
}

static bool is_transpose(const std::vector<float2>& h, int nthreads, int iters) {
    // an odd number of transposes leaves the transpose, an even number the identity
    for (int t = 0; t < nthreads; ++t)
        for (int j = 0; j < 16; ++j) {
            const int g0 = t & ~15, r = t & 15;
            const int src = (iters & 1) ? (g0 + j) * 16 + r : t * 16 + j;
            if (h[(size_t)t * 16 + j].x != (float)src) return false;
        }
    return true;
}

int main() {
    int dev = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int blocks = sms * 8;
    const size_t n = (size_t)blocks * kThreads * 16;
    float2* out = nullptr;
    if (cudaMalloc((void**)&out, n * sizeof(float2)) != cudaSuccess) { printf("{\"error\": \"cudaMalloc\"}\n"); return 1; }
    std::vector<float2> h(n);
    bool ok[2] = {false, false};
    double ms[2] = {0, 0};
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    for (int which = 0; which < 2; ++which) {
        auto run = [&](int iters) { if (which == 0) k_smem<<<blocks, kThreads>>>(out, iters); else k_shfl<<<blocks, kThreads>>>(out, iters); };
        run(1);
        cudaMemcpy(h.data(), out, n * sizeof(float2), cudaMemcpyDeviceToHost);
        ok[which] = is_transpose(h, blocks * kThreads, 1);
        run(kIters);                                       // warm-up
        float best = 1e30f;
        for (int rep = 0; rep < 5; ++rep) {
            cudaEventRecord(e0); run(kIters); cudaEventRecord(e1); cudaEventSynchronize(e1);
            float t = 0; cudaEventElapsedTime(&t, e0, e1);
            if (t < best) best = t;
        }
        ms[which] = best;
    }
    const double elems = (double)n * kIters;
    printf("{\"sms\": %d, \"elements\": %.0f, \"smem_ms\": %.4f, \"shfl_ms\": %.4f, \"smem_ps_per_element\": %.3f, "
           "\"shfl_ps_per_element\": %.3f, \"shfl_over_smem\": %.3f, \"smem_ok\": %s, \"shfl_ok\": %s}\n",
           sms, elems, ms[0], ms[1], ms[0] * 1e9 / elems, ms[1] * 1e9 / elems, ms[1] / ms[0], ok[0] ? "true" : "false",
           ok[1] ? "true" : "false");
    cudaFree(out);
    return (ok[0] && ok[1] && cudaGetLastError() == cudaSuccess) ? 0 : 2;
}
