// link_probe.cu -- standalone measurement program (not part of libconcordia.so): how fast can 512 MiB go from HBM to pinned host
// memory through the copy engine, through SM stores of several flavours and grid sizes, and through bulk (TMA) stores; and
// back.  Build + run: nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o /tmp/link_probe paper_2606_23521_b200/csrc/link_probe.cu && /tmp/link_probe
#include <cstdio>
#include <cstdint>
#include <cuda_runtime.h>
#define CK(x) do { cudaError_t e = (x); if (e != cudaSuccess) { printf("err %s line %d\n", cudaGetErrorString(e), __LINE__); return 1; } } while (0)

__device__ __forceinline__ void st_na(uint4* p, uint4 v) { asm volatile("st.global.L1::no_allocate.v4.u32 [%0], {%1,%2,%3,%4};" :: "l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory"); }
__device__ __forceinline__ void st_cs(uint4* p, uint4 v) { asm volatile("st.global.cs.v4.u32 [%0], {%1,%2,%3,%4};" :: "l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory"); }
__device__ __forceinline__ void st_wt(uint4* p, uint4 v) { asm volatile("st.global.wt.v4.u32 [%0], {%1,%2,%3,%4};" :: "l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory"); }

template <int MODE>
__global__ void k_copy(const uint4* __restrict__ src, uint4* dst, size_t nseg) {   // warp per 4 KiB segment
    const unsigned lane = threadIdx.x & 31;
    const size_t w = (size_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), nw = (size_t)gridDim.x * (blockDim.x >> 5);
    for (size_t s = w; s < nseg; s += nw) {
        uint4 v[8];
#pragma unroll
        for (int u = 0; u < 8; u++) v[u] = src[s * 256 + lane + 32 * u];
#pragma unroll
        for (int u = 0; u < 8; u++) {
            uint4* p = dst + s * 256 + lane + 32 * u;
            if (MODE == 0) st_na(p, v[u]); else if (MODE == 1) *p = v[u]; else if (MODE == 2) st_cs(p, v[u]); else st_wt(p, v[u]);
        }
    }
}

// TMA-style bulk store: stage CH bytes in shared memory per warp-group, one thread issues cp.async.bulk smem -> global
template <int CH>
__global__ void k_bulk(const uint4* __restrict__ src, uint4* dst, size_t nchunks) {
    extern __shared__ __align__(128) unsigned char smem[];
    for (size_t c = blockIdx.x; c < nchunks; c += gridDim.x) {
        uint4* s = reinterpret_cast<uint4*>(smem);
        for (int i = threadIdx.x; i < CH / 16; i += blockDim.x) s[i] = src[c * (CH / 16) + i];
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncthreads();
        if (threadIdx.x == 0) {
            unsigned sa = (unsigned)__cvta_generic_to_shared(smem);
            asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" :: "l"(dst + c * (CH / 16)), "r"(sa), "r"(CH) : "memory");
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
            asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
        }
        __syncthreads();
    }
}

int main() {
    const size_t N = 512ull << 20;
    uint4 *d_src, *h_dst, *d_dst;
    CK(cudaMalloc(&d_src, N)); CK(cudaMemset(d_src, 7, N));
    CK(cudaHostAlloc(&h_dst, N, cudaHostAllocMapped));
    CK(cudaMalloc(&d_dst, N));
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    float ms;
    auto report = [&](const char* name) { cudaEventElapsedTime(&ms, e0, e1); printf("%-44s %8.3f ms  %6.2f GB/s\n", name, ms, N / ms / 1e6); };
    for (int rep = 0; rep < 2; rep++) {
        cudaEventRecord(e0); CK(cudaMemcpyAsync(h_dst, d_src, N, cudaMemcpyDeviceToHost)); cudaEventRecord(e1); CK(cudaDeviceSynchronize()); report("cudaMemcpyAsync D2H (copy engine)");
    }
    const int grids[] = {16, 37, 74, 148, 296, 592, 1184};
    for (int g : grids) {
        char nm[96];
        cudaEventRecord(e0); k_copy<0><<<g, 256>>>(d_src, h_dst, N / 4096); cudaEventRecord(e1); CK(cudaDeviceSynchronize()); snprintf(nm, 96, "st no_allocate v4, grid %d x 256", g); report(nm);
    }
    cudaEventRecord(e0); k_copy<1><<<592, 256>>>(d_src, h_dst, N / 4096); cudaEventRecord(e1); CK(cudaDeviceSynchronize()); report("st default v4, grid 592");
    cudaEventRecord(e0); k_copy<2><<<592, 256>>>(d_src, h_dst, N / 4096); cudaEventRecord(e1); CK(cudaDeviceSynchronize()); report("st .cs v4, grid 592");
    cudaEventRecord(e0); k_copy<3><<<592, 256>>>(d_src, h_dst, N / 4096); cudaEventRecord(e1); CK(cudaDeviceSynchronize()); report("st .wt v4, grid 592");
    for (int g : {37, 148, 592}) {
        char nm[96];
        cudaFuncSetAttribute(k_bulk<16384>, cudaFuncAttributeMaxDynamicSharedMemorySize, 16384);
        cudaEventRecord(e0); k_bulk<16384><<<g, 256, 16384>>>(d_src, h_dst, N / 16384); cudaEventRecord(e1); CK(cudaDeviceSynchronize()); snprintf(nm, 96, "bulk store 16 KiB chunks, grid %d", g); report(nm);
        cudaFuncSetAttribute(k_bulk<65536>, cudaFuncAttributeMaxDynamicSharedMemorySize, 65536);
        cudaEventRecord(e0); k_bulk<65536><<<g, 256, 65536>>>(d_src, h_dst, N / 65536); cudaEventRecord(e1); CK(cudaDeviceSynchronize()); snprintf(nm, 96, "bulk store 64 KiB chunks, grid %d", g); report(nm);
        cudaEventRecord(e0); k_bulk<4096><<<g * 2, 256, 4096>>>(d_src, h_dst, N / 4096); cudaEventRecord(e1); CK(cudaDeviceSynchronize()); snprintf(nm, 96, "bulk store 4 KiB chunks, grid %d", g * 2); report(nm);
    }
    // sanity: bulk store correctness
    unsigned char* hb = (unsigned char*)h_dst; size_t bad = 0; for (size_t i = 0; i < N; i += 4099) bad += hb[i] != 7;
    printf("bad=%zu\n", bad);
    // H2D reads by SM (apply side) for reference
    cudaEventRecord(e0); k_copy<0><<<592, 256>>>(h_dst, d_dst, N / 4096); cudaEventRecord(e1); CK(cudaDeviceSynchronize()); report("SM loads from pinned host -> device, grid 592");
    cudaEventRecord(e0); CK(cudaMemcpyAsync(d_dst, h_dst, N, cudaMemcpyHostToDevice)); cudaEventRecord(e1); CK(cudaDeviceSynchronize()); report("cudaMemcpyAsync H2D (copy engine)");
    return 0;
}
