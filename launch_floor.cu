// launch_floor.cu -- measurement aid beside bench.py (not part of the library): what ONE dependent kernel launch costs
// inside a CUDA graph on this GPU, and what a "last CTA finishes the job" tail (fence + integer ticket + re-read of
// the other CTAs' partials) costs, so that the single-pair latency of iqa_fused_tiles + iqa_aggregate (DESIGN.md
// section 8) can be split into launch floor, DRAM time and the kernels' own ramp and tail.
//   null      empty kernel, grid x 320 threads, same shared-memory footprint class as tma_kernel
//   ticket    every CTA writes a 32-byte partial, __threadfence, atomicAdd on a ticket; the last CTA re-reads all
//             partials with 256 threads, reduces them (shuffles) and writes 8 bytes
// Each number: microseconds per kernel, 64 kernels back to back in one graph, best of 20 replays, with and without
// programmatic dependent launch.   Build: nvcc -O3 -gencode arch=compute_100a,code=sm_100a -o launch_floor launch_floor.cu
#include <cuda_runtime.h>
#include <cstdio>

__global__ void __launch_bounds__(320, 2) null_kernel(int pdl) {
    if (pdl) {
        asm volatile("griddepcontrol.wait;" ::: "memory");
        asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    }
}

__global__ void __launch_bounds__(320, 2) ticket_kernel(int pdl, double4* part, unsigned* ticket, float* out) {
    __shared__ int last;
    __shared__ double4 wsum[10];
    if (pdl) {
        asm volatile("griddepcontrol.wait;" ::: "memory");
        asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    }
    if (threadIdx.x == 0) {
        part[blockIdx.x] = make_double4(1.0, 2.0, 3.0, (double)blockIdx.x);
        __threadfence();
        last = atomicAdd(ticket, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!last) return;
    double4 a = make_double4(0, 0, 0, 0);
    for (unsigned i = threadIdx.x; i < gridDim.x; i += blockDim.x) {
        const double2 q0 = __ldcg(reinterpret_cast<const double2*>(part + i));
        const double2 q1 = __ldcg(reinterpret_cast<const double2*>(part + i) + 1);
        a.x += q0.x; a.y += q0.y; a.z += q1.x; a.w += q1.y;
    }
    for (int o = 16; o > 0; o >>= 1) {
        a.x += __shfl_xor_sync(0xffffffffu, a.x, o); a.y += __shfl_xor_sync(0xffffffffu, a.y, o);
        a.z += __shfl_xor_sync(0xffffffffu, a.z, o); a.w += __shfl_xor_sync(0xffffffffu, a.w, o);
    }
    if ((threadIdx.x & 31) == 0) wsum[threadIdx.x >> 5] = a;
    __syncthreads();
    if (threadIdx.x == 0) {
        double4 s = wsum[0];
        for (int w = 1; w < 10; ++w) { s.x += wsum[w].x; s.y += wsum[w].y; s.z += wsum[w].z; s.w += wsum[w].w; }
        out[0] = (float)(s.x / (s.y + 1e-6));
        out[1] = (float)(s.z / (s.w + 1e-6));
        *ticket = 0u;
    }
}

static float run(bool ticket, int grid, int pdl, int n, double4* part, unsigned* tk, float* out) {
    cudaStream_t st;
    cudaStreamCreate(&st);
    cudaGraph_t g;
    cudaGraphExec_t ge;
    cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal);
    for (int i = 0; i < n; ++i) {
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3(grid);
        cfg.blockDim = dim3(320);
        cfg.stream = st;
        cudaLaunchAttribute a[1];
        a[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        a[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = a;
        cfg.numAttrs = pdl ? 1 : 0;
        if (ticket) cudaLaunchKernelEx(&cfg, ticket_kernel, pdl, part, tk, out);
        else cudaLaunchKernelEx(&cfg, null_kernel, pdl);
    }
    cudaStreamEndCapture(st, &g);
    cudaGraphInstantiate(&ge, g, 0);
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    for (int i = 0; i < 5; ++i) cudaGraphLaunch(ge, st);
    cudaStreamSynchronize(st);
    float best = 1e9f;
    for (int r = 0; r < 20; ++r) {
        cudaEventRecord(e0, st);
        cudaGraphLaunch(ge, st);
        cudaEventRecord(e1, st);
        cudaStreamSynchronize(st);
        float ms;
        cudaEventElapsedTime(&ms, e0, e1);
        if (ms < best) best = ms;
    }
    cudaGraphExecDestroy(ge);
    cudaGraphDestroy(g);
    cudaStreamDestroy(st);
    return best * 1000.f / n;
}

int main() {
    double4* part;
    unsigned* tk;
    float* out;
    cudaMalloc(&part, 4096 * sizeof(double4));
    cudaMalloc(&tk, 4);
    cudaMalloc(&out, 8);
    cudaMemset(tk, 0, 4);
    for (int pdl = 0; pdl < 2; ++pdl)
        for (int grid : {1, 148, 296})
            printf("pdl=%d grid=%d: null %.3f us, ticket %.3f us per kernel\n", pdl, grid,
                   run(false, grid, pdl, 64, part, tk, out), run(true, grid, pdl, 64, part, tk, out));
    return cudaDeviceSynchronize() == cudaSuccess ? 0 : 1;
}
