// scan_probe.cu -- standalone measurement program (not part of libconcordia.so): the dirty scan's memory path.
// BASELINE.json's north_star names "TMA or cp.async bulk staging of page tiles into shared memory" as an option for
// the scanner; this program measures that option against the register path cc_scan_kernel uses, on the same job
// (compare two 8 GiB arrays, 16-byte granularity, one flag per 64 KiB page):
//   ldg      warp per 4 KiB segment, 8 + 8 independent ld.global.nc.L1::no_allocate.v4 per lane (cc_scan_kernel's loop)
//   bulk     persistent CTAs, one elected thread issues cp.async.bulk (TMA 1-D) of TILE bytes of each array into a
//            STAGES-deep shared-memory ring (mbarrier complete_tx), all warps compare out of shared memory
// Build + run: nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o /tmp/scan_probe paper_2606_23521_b200/csrc/scan_probe.cu && /tmp/scan_probe
#include <cstdio>
#include <cstdint>
#include <cuda_runtime.h>
#define CK(x) do { cudaError_t e = (x); if (e != cudaSuccess) { printf("err %s line %d\n", cudaGetErrorString(e), __LINE__); return 1; } } while (0)

__device__ __forceinline__ uint4 ld_stream(const uint4* p) {
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}

__global__ void __launch_bounds__(256) k_ldg(const uint4* __restrict__ a, const uint4* __restrict__ b, size_t nseg, unsigned* bitmap) {
    const unsigned lane = threadIdx.x & 31;
    const size_t w = (size_t)blockIdx.x * 8 + (threadIdx.x >> 5), nw = (size_t)gridDim.x * 8;
    for (size_t s = w; s < nseg; s += nw) {
        uint4 va[8], vb[8];
#pragma unroll
        for (int u = 0; u < 8; u++) va[u] = ld_stream(a + s * 256 + lane + 32 * u);
#pragma unroll
        for (int u = 0; u < 8; u++) vb[u] = ld_stream(b + s * 256 + lane + 32 * u);
        unsigned acc = 0;
#pragma unroll
        for (int u = 0; u < 8; u++) acc |= (va[u].x ^ vb[u].x) | (va[u].y ^ vb[u].y) | (va[u].z ^ vb[u].z) | (va[u].w ^ vb[u].w);
        if (__any_sync(0xFFFFFFFFu, acc != 0) && lane == 0) atomicOr(&bitmap[(s >> 4) >> 5], 1u << ((s >> 4) & 31));
    }
}

__device__ __forceinline__ void mbar_init(uint64_t* m, unsigned n) { asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"((unsigned)__cvta_generic_to_shared(m)), "r"(n)); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t* m, unsigned bytes) { asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"((unsigned)__cvta_generic_to_shared(m)), "r"(bytes) : "memory"); }
__device__ __forceinline__ void mbar_arrive(uint64_t* m) { asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" :: "r"((unsigned)__cvta_generic_to_shared(m)) : "memory"); }
__device__ __forceinline__ void mbar_wait(uint64_t* m, unsigned parity) {
    asm volatile("{\n.reg .pred p;\nW: mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n@p bra D;\nbra W;\nD:\n}" :: "r"((unsigned)__cvta_generic_to_shared(m)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_load(void* smem, const void* gmem, unsigned bytes, uint64_t* m) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 :: "r"((unsigned)__cvta_generic_to_shared(smem)), "l"(gmem), "r"(bytes), "r"((unsigned)__cvta_generic_to_shared(m)) : "memory");
}

template <int TILE, int STAGES>
__global__ void __launch_bounds__(256) k_bulk(const unsigned char* __restrict__ a, const unsigned char* __restrict__ b, size_t ntiles, unsigned* bitmap) {
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ uint64_t full[STAGES], empty[STAGES];
    unsigned char* sa = smem;
    unsigned char* sb = smem + (size_t)TILE * STAGES;
    const unsigned tid = threadIdx.x, lane = tid & 31;
    if (tid == 0) {
        for (int s = 0; s < STAGES; s++) { mbar_init(&full[s], 1); mbar_init(&empty[s], 8); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const size_t my = (ntiles > blockIdx.x) ? (ntiles - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
    // prologue: fill the ring
    if (tid == 0)
        for (size_t i = 0; i < my && i < STAGES; i++) {
            const size_t t = blockIdx.x + i * gridDim.x;
            mbar_expect_tx(&full[i], 2 * TILE);
            bulk_load(sa + i * TILE, a + t * TILE, TILE, &full[i]);
            bulk_load(sb + i * TILE, b + t * TILE, TILE, &full[i]);
        }
    for (size_t i = 0; i < my; i++) {
        const int s = (int)(i % STAGES);
        const unsigned ph = (unsigned)((i / STAGES) & 1);
        mbar_wait(&full[s], ph);
        const uint4* pa = reinterpret_cast<const uint4*>(sa + s * TILE);
        const uint4* pb = reinterpret_cast<const uint4*>(sb + s * TILE);
        unsigned acc = 0;
#pragma unroll
        for (int j = 0; j < TILE / 16 / 256; j++) {
            const uint4 x = pa[tid + 256 * j], y = pb[tid + 256 * j];
            acc |= (x.x ^ y.x) | (x.y ^ y.y) | (x.z ^ y.z) | (x.w ^ y.w);
        }
        const bool any = __any_sync(0xFFFFFFFFu, acc != 0);
        const size_t t = blockIdx.x + i * gridDim.x;
        if (any && lane == 0) { const size_t page = t * TILE / 65536; atomicOr(&bitmap[page >> 5], 1u << (page & 31)); }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[s]);                  // this warp is done with the stage
        if (tid == 0 && i + STAGES < my) {                       // refill the stage once all 8 warps have left it
            mbar_wait(&empty[s], ph);
            const size_t tn = blockIdx.x + (i + STAGES) * gridDim.x;
            mbar_expect_tx(&full[s], 2 * TILE);
            bulk_load(sa + s * TILE, a + tn * TILE, TILE, &full[s]);
            bulk_load(sb + s * TILE, b + tn * TILE, TILE, &full[s]);
        }
    }
}

template <int TILE, int STAGES>
static int run_bulk(const unsigned char* a, const unsigned char* b, size_t N, unsigned* bm, int ctas_per_sm, cudaEvent_t e0, cudaEvent_t e1) {
    const size_t smem = (size_t)2 * TILE * STAGES;
    CK(cudaFuncSetAttribute(k_bulk<TILE, STAGES>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    float best = 1e9f;
    for (int r = 0; r < 5; r++) {
        cudaEventRecord(e0);
        k_bulk<TILE, STAGES><<<148 * ctas_per_sm, 256, smem>>>(a, b, N / TILE, bm);
        cudaEventRecord(e1);
        CK(cudaDeviceSynchronize());
        float ms; cudaEventElapsedTime(&ms, e0, e1);
        if (r && ms < best) best = ms;
    }
    printf("bulk  tile %3d KiB x %2d stages, %d CTA/SM (%3zu KiB smem/SM in flight)   %7.3f ms  %7.1f GB/s\n", TILE >> 10, STAGES, ctas_per_sm,
           smem * ctas_per_sm >> 10, best, 2.0 * N / best / 1e6);
    return 0;
}

int main() {
    const size_t N = 8ull << 30;
    unsigned char *a, *b; unsigned* bm;
    CK(cudaMalloc(&a, N)); CK(cudaMalloc(&b, N)); CK(cudaMalloc(&bm, 1 << 20));
    CK(cudaMemset(a, 3, N)); CK(cudaMemset(b, 3, N)); CK(cudaMemset(bm, 0, 1 << 20));
    CK(cudaMemset(a + (5ull << 30) + 12345, 9, 1));                       // one dirty page
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    for (int bps : {2, 3, 4, 5, 6, 8}) {
        float best = 1e9f;
        for (int r = 0; r < 5; r++) {
            cudaEventRecord(e0);
            k_ldg<<<148 * bps, 256>>>((const uint4*)a, (const uint4*)b, N / 4096, bm);
            cudaEventRecord(e1);
            CK(cudaDeviceSynchronize());
            float ms; cudaEventElapsedTime(&ms, e0, e1);
            if (r && ms < best) best = ms;
        }
        printf("ldg   warp per 4 KiB, %d CTA/SM of 256 threads                              %7.3f ms  %7.1f GB/s\n", bps, best, 2.0 * N / best / 1e6);
    }
    if (run_bulk<8192, 6>(a, b, N, bm, 2, e0, e1)) return 1;
    if (run_bulk<16384, 3>(a, b, N, bm, 2, e0, e1)) return 1;
    if (run_bulk<16384, 6>(a, b, N, bm, 1, e0, e1)) return 1;
    if (run_bulk<32768, 3>(a, b, N, bm, 1, e0, e1)) return 1;
    if (run_bulk<16384, 2>(a, b, N, bm, 3, e0, e1)) return 1;
    if (run_bulk<8192, 3>(a, b, N, bm, 4, e0, e1)) return 1;
    unsigned h[4]; CK(cudaMemcpy(h, bm + ((5ull << 30) / 65536 >> 5), 4, cudaMemcpyDeviceToHost));
    unsigned total = 0; { static unsigned hb[1 << 18]; CK(cudaMemcpy(hb, bm, 1 << 20, cudaMemcpyDeviceToHost)); for (unsigned x : hb) total += __builtin_popcount(x); }
    printf("dirty pages found: %u (expected 1)\n", total);
    return 0;
}
