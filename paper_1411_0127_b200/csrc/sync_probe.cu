// sync_probe.cu -- what does it cost to make one half-sweep wait for the previous one on this part?  (DESIGN.md section 6,
// "launch floor"; csrc/persistent.cuh.)  A standalone program (no library code): loops of 2000 synchronisations, CUDA events.
//   grid_barrier: counter in global memory, red.release + ld.acquire polling (variant 0), without the fences (1), with a store of
//                 every thread before each barrier (2); cooperative groups' grid.sync(); a ring of flags handed from CTA to CTA
//                 (st.release / ld.acquire, the pattern of persistent_site_packed); cluster.sync() of one 8-CTA cluster.
//   build + run:  python -m paper_1411_0127_b200.sync_probe
#include <cuda_runtime.h>
#include <cooperative_groups.h>
#include <cstdio>
#include <cstdint>

namespace cg = cooperative_groups;

__device__ __forceinline__ void grid_barrier(unsigned int *counter, unsigned int &target)
{
    target += gridDim.x;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned int v;
        asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(counter) : "memory");
        do { asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(counter) : "memory"); } while ((int)(v - target) < 0);
    }
    __syncthreads();
}
// relaxed variant: no fences at all (only latency of atomic + poll)
__device__ __forceinline__ void grid_barrier_relaxed(unsigned int *counter, unsigned int &target)
{
    target += gridDim.x;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned int v;
        asm volatile("red.relaxed.gpu.global.add.u32 [%0], 1;" ::"l"(counter) : "memory");
        do { asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(counter) : "memory"); } while ((int)(v - target) < 0);
    }
    __syncthreads();
}
__global__ void k_bar(unsigned int *ctr, int n, int variant, uint32_t *data)
{
    unsigned int target = 0;
    for (int i = 0; i < n; ++i) {
        if (variant == 2) data[blockIdx.x * blockDim.x + threadIdx.x] = i;   // a store before each barrier
        if (variant == 1) grid_barrier_relaxed(ctr, target); else grid_barrier(ctr, target);
    }
}
__global__ void k_cg(int n)
{
    cg::grid_group g = cg::this_grid();
    for (int i = 0; i < n; ++i) g.sync();
}
// ring of flags: CTA b waits for flag[b-1] >= i+1 (and flag[b+1]) then publishes its own flag = i+1 after storing data: dataflow
__global__ void k_flags(unsigned int *flag, int n, uint32_t *data, int dostore)
{
    const int b = blockIdx.x, G = gridDim.x;
    const int l = (b + G - 1) % G, r = (b + 1) % G;
    for (int i = 1; i <= n; ++i) {
        if (dostore) data[b * blockDim.x + threadIdx.x] = i;
        __syncthreads();
        if (threadIdx.x == 0) asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(flag + b * 32), "r"(i) : "memory");
        if (threadIdx.x < 2) {
            unsigned int v;
            const unsigned int *p = flag + (threadIdx.x ? r : l) * 32;
            do { asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory"); } while ((int)(v - i) < 0);
        }
        __syncthreads();
    }
}
__global__ void __cluster_dims__(8, 1, 1) k_cluster(int n)
{
    cg::cluster_group c = cg::this_cluster();
    for (int i = 0; i < n; ++i) c.sync();
}
// launch floor: empty (and 1 us) kernels launched into a stream, plainly and with programmatic stream serialization, and replayed
// from an instantiated graph of 200 nodes
__global__ void k_empty(int *p) { asm volatile("griddepcontrol.wait;" ::: "memory"); if (p && threadIdx.x == 1000) *p = 1; }
__global__ void k_work(int *p, int n)
{
    asm volatile("griddepcontrol.wait;" ::: "memory");
    int v = threadIdx.x;
    for (int i = 0; i < n; ++i) v = v * 1664525 + 1013904223;
    if (v == 12345) *p = v;
}
template <typename... A> void launch_pdl(void (*k)(A...), dim3 g, dim3 b, cudaStream_t st, A... a)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = g; cfg.blockDim = b; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    cudaLaunchKernelEx(&cfg, k, a...);
}
static void launch_floor()
{
    int *d; cudaMalloc(&d, 4);
    cudaStream_t st; cudaStreamCreate(&st);
    cudaEvent_t a, b; cudaEventCreate(&a); cudaEventCreate(&b);
    const int N = 20000;
    const char *names[4] = {"stream launch, empty kernel", "stream launch + programmatic dependent launch, empty kernel",
                            "stream launch + programmatic dependent launch, 1 us kernel", "graph of 200 empty kernels, replayed"};
    for (int mode = 0; mode < 4; ++mode) for (int grid : {16, 148, 1024}) {
        for (int i = 0; i < 100; ++i) k_empty<<<grid, 128, 0, st>>>(d);
        cudaStreamSynchronize(st);
        cudaEventRecord(a, st);
        if (mode == 0) for (int i = 0; i < N; ++i) k_empty<<<grid, 128, 0, st>>>(d);
        if (mode == 1) for (int i = 0; i < N; ++i) launch_pdl(k_empty, dim3(grid), dim3(128), st, d);
        if (mode == 2) for (int i = 0; i < N; ++i) launch_pdl(k_work, dim3(grid), dim3(128), st, d, 2000);
        if (mode == 3) {
            cudaGraph_t g; cudaGraphExec_t ge;
            cudaStreamBeginCapture(st, cudaStreamCaptureModeGlobal);
            for (int i = 0; i < 200; ++i) k_empty<<<grid, 128, 0, st>>>(d);
            cudaStreamEndCapture(st, &g); cudaGraphInstantiate(&ge, g, 0);
            cudaEventRecord(a, st);
            for (int i = 0; i < N / 200; ++i) cudaGraphLaunch(ge, st);
        }
        cudaEventRecord(b, st); cudaEventSynchronize(b);
        float ms; cudaEventElapsedTime(&ms, a, b);
        printf("%-64s grid %4d x 128 threads: %.3f us per kernel\n", names[mode], grid, 1e3 * ms / N);
    }
}

int main()
{
    launch_floor();
    unsigned int *ctr; uint32_t *data; unsigned int *flag;
    cudaMalloc(&ctr, 4); cudaMalloc(&data, 4 * 2048 * 1024); cudaMalloc(&flag, 4 * 32 * 4096);
    cudaEvent_t a, b; cudaEventCreate(&a); cudaEventCreate(&b);
    const int n = 2000;
    for (int threads : {256}) for (int G : {1, 16, 148, 296, 592, 1184}) {
        for (int variant = 0; variant < 3; ++variant) {
            cudaMemset(ctr, 0, 4);
            void *args[] = {&ctr, (void *)&n, &variant, &data};
            cudaEventRecord(a);
            cudaError_t e = cudaLaunchCooperativeKernel((const void *)k_bar, dim3(G), dim3(threads), args, 0, 0);
            cudaEventRecord(b); cudaEventSynchronize(b);
            float ms; cudaEventElapsedTime(&ms, a, b);
            printf("grid_barrier variant %d (0 rel/acq, 1 relaxed, 2 rel/acq + store)  G=%4d thr=%d : %.3f us per barrier  (%s)\n", variant, G, threads, 1e3 * ms / n, cudaGetErrorString(e));
        }
        {
            void *args[] = {(void *)&n};
            cudaEventRecord(a);
            cudaError_t e = cudaLaunchCooperativeKernel((const void *)k_cg, dim3(G), dim3(threads), args, 0, 0);
            cudaEventRecord(b); cudaEventSynchronize(b);
            float ms; cudaEventElapsedTime(&ms, a, b);
            printf("cg grid.sync                                   G=%4d thr=%d : %.3f us per barrier  (%s)\n", G, threads, 1e3 * ms / n, cudaGetErrorString(e));
        }
        for (int dostore = 0; dostore < 2; ++dostore) {
            cudaMemset(flag, 0, 4 * 32 * 4096);
            void *args[] = {&flag, (void *)&n, &data, &dostore};
            cudaEventRecord(a);
            cudaError_t e = cudaLaunchCooperativeKernel((const void *)k_flags, dim3(G), dim3(threads), args, 0, 0);
            cudaEventRecord(b); cudaEventSynchronize(b);
            float ms; cudaEventElapsedTime(&ms, a, b);
            printf("neighbour flags (store=%d)                      G=%4d thr=%d : %.3f us per step     (%s)\n", dostore, G, threads, 1e3 * ms / n, cudaGetErrorString(e));
        }
    }
    {
        cudaEventRecord(a);
        k_cluster<<<8, 256>>>(n);
        cudaEventRecord(b); cudaEventSynchronize(b);
        float ms; cudaEventElapsedTime(&ms, a, b);
        printf("cluster.sync, one cluster of 8 CTAs x 256: %.3f us per sync (%s)\n", 1e3 * ms / n, cudaGetErrorString(cudaGetLastError()));
    }
    return 0;
}
