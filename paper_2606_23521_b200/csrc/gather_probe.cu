// gather_probe.cu -- one-off measurement: the record writer's memory path on an all-dirty region.
// Job: for every page p of an N-byte region (page P): log[p*(P+16)+16 ..] = shadow[p*P ..] = base[p*P ..]   (1 read, 2 writes)
//   reg     warp per 4 KiB segment: 8 x ld.v4 -> 8 x st.v4 (log) + 8 x st.v4 (shadow)            (cc_gather_items' loop, no CRC)
//   bulk    one thread per CTA drives a ring of STAGES tiles: cp.async.bulk global->shared (mbarrier complete_tx), then two
//           cp.async.bulk shared->global (log, shadow) per tile; no consumer warps (pure DMA)
//   bulkcrc the same ring, plus consumer warps that read the tile out of shared memory and run the library's CRC over it
// nvcc -gencode arch=compute_100a,code=sm_100a -O3 -std=c++17 -I paper_2606_23521_b200/csrc -o /tmp/gather_probe paper_2606_23521_b200/csrc/gather_probe.cu && /tmp/gather_probe 8
#include <cstdio>
#include <cstdint>
#include <cuda_runtime.h>
#include "cc_common.cuh"
#include "cc_crc.cuh"
#define CK(x) do { cudaError_t e = (x); if (e != cudaSuccess) { printf("err %s line %d\n", cudaGetErrorString(e), __LINE__); return 1; } } while (0)

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
__device__ __forceinline__ void bulk_store(void* gmem, const void* smem, unsigned bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" :: "l"(gmem), "r"((unsigned)__cvta_generic_to_shared(smem)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read %0;" :: "n"(N) : "memory"); }
template <int N> __device__ __forceinline__ void bulk_wait() { asm volatile("cp.async.bulk.wait_group %0;" :: "n"(N) : "memory"); }

// ---- register path ----
template <int NDST>
__global__ void __launch_bounds__(256) k_reg(const u8* __restrict__ base, u8* shadow, u8* log, size_t nseg, u32 P, u32 hdr) {
    const unsigned lane = threadIdx.x & 31;
    const size_t w = (size_t)blockIdx.x * 8 + (threadIdx.x >> 5), nw = (size_t)gridDim.x * 8;
    const u32 spp = P / 4096;
    for (size_t s = w; s < nseg; s += nw) {
        const size_t p = s / spp, c = s % spp;
        const uint4* src = reinterpret_cast<const uint4*>(base + s * 4096);
        uint4* d1 = reinterpret_cast<uint4*>(log + p * ((size_t)P + hdr) + hdr + c * 4096);
        uint4* d2 = reinterpret_cast<uint4*>(shadow + s * 4096);
        uint4 v[8];
#pragma unroll
        for (int u = 0; u < 8; u++) v[u] = ld_stream(src + lane + 32 * u);
#pragma unroll
        for (int u = 0; u < 8; u++) st_stream(d1 + lane + 32 * u, v[u]);
        if (NDST == 2) {
#pragma unroll
            for (int u = 0; u < 8; u++) st_stream(d2 + lane + 32 * u, v[u]);
        }
    }
}

// ---- register path, log stores rotated across lanes so that every warp-wide store instruction starts on a 16*MOD-byte boundary ----
template <int MOD>
__global__ void __launch_bounds__(256) k_reg_shift(const u8* __restrict__ base, u8* shadow, u8* log, size_t nseg, u32 P, u32 hdr) {
    const unsigned lane = threadIdx.x & 31;
    const size_t w = (size_t)blockIdx.x * 8 + (threadIdx.x >> 5), nw = (size_t)gridDim.x * 8;
    const u32 spp = P / 4096;
    for (size_t s = w; s < nseg; s += nw) {
        const size_t p = s / spp, c = s % spp;
        const uint4* src = reinterpret_cast<const uint4*>(base + s * 4096);
        uint4* d1 = reinterpret_cast<uint4*>(log + p * ((size_t)P + hdr) + hdr + c * 4096);
        uint4* d2 = reinterpret_cast<uint4*>(shadow + s * 4096);
        const u32 a = (u32)((reinterpret_cast<uintptr_t>(d1) >> 4) & (MOD - 1));   // vectors past the last boundary
        uint4 v[8];
#pragma unroll
        for (int u = 0; u < 8; u++) v[u] = ld_stream(src + lane + 32 * u);
#pragma unroll
        for (int u = 0; u < 8; u++) st_stream(d2 + lane + 32 * u, v[u]);
        // log: instruction u stores vectors [32u - a, 32u - a + 32): lane l holds lane (l - a)'s vector
        const u32 from = (lane - a) & 31u;
        uint4 prev = make_uint4(0, 0, 0, 0);
#pragma unroll
        for (int u = 0; u < 8; u++) {
            uint4 r;
            r.x = __shfl_sync(0xFFFFFFFFu, v[u].x, from); r.y = __shfl_sync(0xFFFFFFFFu, v[u].y, from);
            r.z = __shfl_sync(0xFFFFFFFFu, v[u].z, from); r.w = __shfl_sync(0xFFFFFFFFu, v[u].w, from);
            const uint4 o = lane >= a ? r : prev;            // lanes < a: the tail of the previous 512 bytes
            if (u > 0 || lane >= a) st_stream(d1 + (32 * u + (int)lane - (int)a), o);
            prev = r;
        }
        if (lane < a) st_stream(d1 + (256 + (int)lane - (int)a), prev);
    }
}

// ---- bulk path, pure DMA: 32-thread CTAs, lane 0 drives the ring ----
template <int NDST>
__global__ void __launch_bounds__(32) k_bulk(const u8* __restrict__ base, u8* shadow, u8* log, size_t ntiles, u32 P, u32 hdr, u32 TILE, u32 STAGES) {
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ uint64_t full[16];
    if (threadIdx.x != 0) return;
    for (u32 s = 0; s < STAGES; s++) mbar_init(&full[s], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    const size_t my = (ntiles > blockIdx.x) ? (ntiles - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
    const u32 tpp = P / TILE;
    for (size_t i = 0; i < my && i < STAGES; i++) {
        const size_t t = blockIdx.x + i * gridDim.x;
        mbar_expect_tx(&full[i], TILE);
        bulk_load(smem + i * TILE, base + t * TILE, TILE, &full[i]);
    }
    for (size_t i = 0; i < my; i++) {
        const u32 s = (u32)(i % STAGES);
        mbar_wait(&full[s], (u32)((i / STAGES) & 1));
        const size_t t = blockIdx.x + i * gridDim.x;
        const size_t p = t / tpp, c = t % tpp;
        bulk_store(log + p * ((size_t)P + hdr) + hdr + c * TILE, smem + s * TILE, TILE);
        if (NDST == 2) bulk_store(shadow + t * TILE, smem + s * TILE, TILE);
        bulk_commit();
        if (i >= 1 && i - 1 + STAGES < my) {          // refill the previous tile's stage once its stores have read it
            bulk_wait_read<1>();
            const u32 sp = (u32)((i - 1) % STAGES);
            const size_t tn = blockIdx.x + (i - 1 + STAGES) * gridDim.x;
            mbar_expect_tx(&full[sp], TILE);
            bulk_load(smem + sp * TILE, base + tn * TILE, TILE, &full[sp]);
        }
    }
    bulk_wait<0>();
}

// ---- bulk path + CRC by consumer warps: CTA of (1 + NW) warps; warp 0 lane 0 = DMA, warps 1..NW = CRC over 4 KiB segments of the tile
struct probe_smem_ctl { uint64_t full[8]; uint64_t empty[8]; };
template <int NW>
__global__ void __launch_bounds__(32 * (NW + 1)) k_bulkcrc(const u8* __restrict__ base, u8* shadow, u8* log, size_t ntiles, u32 P, u32 hdr, u32 TILE,
                                                            u32 STAGES, const cc_crc_tables* tabs, u32* crc_out) {
    extern __shared__ __align__(128) unsigned char smem[];
    cc_crc_smem* cs = reinterpret_cast<cc_crc_smem*>(smem);
    u8* ring = smem + ((sizeof(cc_crc_smem) + 127) / 128) * 128;
    __shared__ probe_smem_ctl ctl;
    const u32 tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    if (tid == 0) {
        for (u32 s = 0; s < STAGES; s++) { mbar_init(&ctl.full[s], 1); mbar_init(&ctl.empty[s], NW); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    cc_crc_smem_init(cs, tabs);       // (has a __syncthreads at its end)
    const size_t my = (ntiles > blockIdx.x) ? (ntiles - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
    const u32 tpp = P / TILE;
    if (wid == 0) {
        if (lane != 0) return;
        for (size_t i = 0; i < my && i < STAGES; i++) {
            const size_t t = blockIdx.x + i * gridDim.x;
            mbar_expect_tx(&ctl.full[i], TILE);
            bulk_load(ring + i * TILE, base + t * TILE, TILE, &ctl.full[i]);
        }
        for (size_t i = 0; i < my; i++) {
            const u32 s = (u32)(i % STAGES);
            mbar_wait(&ctl.full[s], (u32)((i / STAGES) & 1));
            const size_t t = blockIdx.x + i * gridDim.x;
            const size_t p = t / tpp, c = t % tpp;
            bulk_store(log + p * ((size_t)P + hdr) + hdr + c * TILE, ring + s * TILE, TILE);
            bulk_store(shadow + t * TILE, ring + s * TILE, TILE);
            bulk_commit();
            if (i >= 1 && i - 1 + STAGES < my) {
                const u32 sp = (u32)((i - 1) % STAGES);
                bulk_wait_read<1>();
                mbar_wait(&ctl.empty[sp], (u32)(((i - 1) / STAGES) & 1));      // the CRC warps have left it too
                const size_t tn = blockIdx.x + (i - 1 + STAGES) * gridDim.x;
                mbar_expect_tx(&ctl.full[sp], TILE);
                bulk_load(ring + sp * TILE, base + tn * TILE, TILE, &ctl.full[sp]);
            }
        }
        bulk_wait<0>();
        return;
    }
    const u32 cw = wid - 1;
    const u32 segs = TILE / 4096;
    u32 accum = 0;
    for (size_t i = 0; i < my; i++) {
        const u32 s = (u32)(i % STAGES);
        mbar_wait(&ctl.full[s], (u32)((i / STAGES) & 1));
        for (u32 g = cw; g < segs; g += NW) {
            const uint4* sp = reinterpret_cast<const uint4*>(ring + s * TILE + g * 4096);
            uint4 v[8];
#pragma unroll
            for (int u = 0; u < 8; u++) v[u] = sp[lane + 32 * u];
            accum ^= crc_segment_warp<8>(cs, tabs, v, 256, 0, lane);
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&ctl.empty[s]);
    }
    if (lane == 0 && accum == 0x12345678u) crc_out[0] = accum;
}

// ---- register path + CRC (the library's loop) ----
__global__ void __launch_bounds__(256, 4) k_regcrc(const u8* __restrict__ base, u8* shadow, u8* log, size_t nseg, u32 P, u32 hdr,
                                                  const cc_crc_tables* tabs, u32* crc_out) {
    extern __shared__ __align__(128) unsigned char smem[];
    cc_crc_smem* cs = reinterpret_cast<cc_crc_smem*>(smem);
    cc_crc_smem_init(cs, tabs);
    const unsigned lane = threadIdx.x & 31;
    const size_t w = (size_t)blockIdx.x * 8 + (threadIdx.x >> 5), nw = (size_t)gridDim.x * 8;
    const u32 spp = P / 4096;
    u32 accum = 0;
    for (size_t s = w; s < nseg; s += nw) {
        const size_t p = s / spp, c = s % spp;
        const uint4* src = reinterpret_cast<const uint4*>(base + s * 4096);
        uint4* d1 = reinterpret_cast<uint4*>(log + p * ((size_t)P + hdr) + hdr + c * 4096);
        uint4* d2 = reinterpret_cast<uint4*>(shadow + s * 4096);
        uint4 v[8];
#pragma unroll
        for (int u = 0; u < 8; u++) v[u] = ld_stream(src + lane + 32 * u);
#pragma unroll
        for (int u = 0; u < 8; u++) st_stream(d1 + lane + 32 * u, v[u]);
#pragma unroll
        for (int u = 0; u < 8; u++) st_stream(d2 + lane + 32 * u, v[u]);
        accum ^= crc_segment_warp<8>(cs, tabs, v, 256, 0, lane);
    }
    if (lane == 0 && accum == 0x12345678u) crc_out[0] = accum;
}

__global__ void k_check(const u8* base, const u8* shadow, const u8* log, size_t nvec, u32 P, u32 hdr, unsigned long long* bad) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += (size_t)gridDim.x * blockDim.x) {
        const size_t off = i * 16, p = off / P, o = off % P;
        const uint4 a = *reinterpret_cast<const uint4*>(base + off);
        const uint4 b = *reinterpret_cast<const uint4*>(shadow + off);
        const uint4 c = *reinterpret_cast<const uint4*>(log + p * ((size_t)P + hdr) + hdr + o);
        if (a.x != b.x || a.y != b.y || a.z != b.z || a.w != b.w || a.x != c.x || a.y != c.y || a.z != c.z || a.w != c.w) atomicAdd(bad, 1ull);
    }
}
__global__ void k_fill(u32* p, size_t n, u32 seed) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        u32 x = (u32)i * 2654435761u ^ seed; x ^= x >> 15; x *= 2246822519u; x ^= x >> 13;
        p[i] = x;
    }
}

static cudaEvent_t e0, e1;
template <typename F> static float time_best(F f, int reps = 5) {
    float best = 1e9f;
    for (int r = 0; r < reps; r++) {
        cudaEventRecord(e0); f(); cudaEventRecord(e1);
        cudaDeviceSynchronize();
        float ms; cudaEventElapsedTime(&ms, e0, e1);
        if (r && ms < best) best = ms;
    }
    return best;
}

int main(int argc, char** argv) {
    const size_t N = (argc > 1 ? (size_t)atoi(argv[1]) : 8) << 30;
    u8 *base, *shadow, *log; unsigned long long* bad; u32* crc_out; cc_crc_tables* d_tabs;
    CK(cudaMalloc(&base, N)); CK(cudaMalloc(&shadow, N)); CK(cudaMalloc(&log, N + N / 4096 * 16 + 4096));
    CK(cudaMalloc(&bad, 8)); CK(cudaMalloc(&crc_out, 8)); CK(cudaMalloc(&d_tabs, sizeof(cc_crc_tables)));
    static cc_crc_tables h_tabs; cc_crc_build_tables(&h_tabs);
    CK(cudaMemcpy(d_tabs, &h_tabs, sizeof(h_tabs), cudaMemcpyHostToDevice));
    k_fill<<<148 * 8, 256>>>((u32*)base, N / 4, 12345u);
    CK(cudaDeviceSynchronize());
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    auto check = [&](u32 P, u32 hdr, const char* what) -> int {
        cudaMemset(bad, 0, 8);
        k_check<<<148 * 8, 256>>>(base, shadow, log, N / 16, P, hdr, bad);
        unsigned long long h = 0; cudaMemcpy(&h, bad, 8, cudaMemcpyDeviceToHost);
        if (h) printf("   !! %s: %llu mismatching vectors\n", what, h);
        cudaMemset(shadow, 0, N); cudaMemset(log, 0, N + N / 4096 * 16);
        return (int)(h != 0);
    };
    {   // reference: cudaMemcpy D2D (1R + 1W)
        float ms = time_best([&] { cudaMemcpyAsync(shadow, base, N, cudaMemcpyDeviceToDevice); });
        printf("cudaMemcpy D2D (1R+1W)                                              %8.3f ms  %7.1f GB/s\n", ms, 2.0 * N / ms / 1e6);
    }
    for (u32 P : {65536u, 4096u}) {
        for (u32 hdr : {16u, 0u}) {
            printf("---- P = %u KiB, record header %u bytes, N = %zu GiB\n", P >> 10, hdr, N >> 30);
            for (int bps : {2, 4, 6, 8}) {
                float ms = time_best([&] { k_reg<2><<<148 * bps, 256>>>(base, shadow, log, N / 4096, P, hdr); });
                printf("reg   1R+2W, %d CTA/SM x 256 thr                                      %8.3f ms  %7.1f GB/s\n", bps, ms, 3.0 * N / ms / 1e6);
                check(P, hdr, "reg");
            }
            for (int bps : {4, 5}) {
                float ms = time_best([&] { k_reg_shift<2><<<148 * bps, 256>>>(base, shadow, log, N / 4096, P, hdr); });
                printf("reg-shift(32 B) 1R+2W, %d CTA/SM x 256 thr                              %8.3f ms  %7.1f GB/s\n", bps, ms, 3.0 * N / ms / 1e6);
                check(P, hdr, "regshift2");
                ms = time_best([&] { k_reg_shift<8><<<148 * bps, 256>>>(base, shadow, log, N / 4096, P, hdr); });
                printf("reg-shift(128 B) 1R+2W, %d CTA/SM x 256 thr                             %8.3f ms  %7.1f GB/s\n", bps, ms, 3.0 * N / ms / 1e6);
                check(P, hdr, "regshift8");
            }
            {
                float ms = time_best([&] { k_reg<1><<<148 * 6, 256>>>(base, shadow, log, N / 4096, P, hdr); });
                printf("reg   1R+1W (log only), 6 CTA/SM                                      %8.3f ms  %7.1f GB/s\n", ms, 2.0 * N / ms / 1e6);
            }
            if (hdr == 16) {
                CK(cudaFuncSetAttribute(k_regcrc, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(cc_crc_smem)));
                float ms = time_best([&] { k_regcrc<<<148 * 4, 256, sizeof(cc_crc_smem)>>>(base, shadow, log, N / 4096, P, hdr, d_tabs, crc_out); });
                printf("reg+crc 1R+2W, 4 CTA/SM x 256 thr (library loop)                       %8.3f ms  %7.1f GB/s\n", ms, 3.0 * N / ms / 1e6);
                check(P, hdr, "regcrc");
            }
            struct V { u32 tile, stages, cps; };
            const V vs[] = {{4096, 4, 8}, {4096, 8, 6}, {8192, 4, 6}, {16384, 3, 4}, {16384, 4, 3}, {32768, 3, 2}, {65536, 3, 1}, {4096, 2, 16}, {8192, 2, 12}, {16384, 2, 6}};
            for (const V& v : vs) {
                if (v.tile > P) continue;
                const size_t sm = (size_t)v.tile * v.stages;
                CK(cudaFuncSetAttribute(k_bulk<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
                float ms = time_best([&] { k_bulk<2><<<148 * v.cps, 32, sm>>>(base, shadow, log, N / v.tile, P, hdr, v.tile, v.stages); });
                printf("bulk  1R+2W, tile %2u KiB x %u stages, %2u CTA/SM (%3zu KiB/SM)            %8.3f ms  %7.1f GB/s\n", v.tile >> 10, v.stages, v.cps,
                       sm * v.cps >> 10, ms, 3.0 * N / ms / 1e6);
                if (cudaGetLastError() != cudaSuccess) printf("   launch error\n");
                check(P, hdr, "bulk");
            }
            if (P >= 16384) {
                const size_t sm = 16384 * 3;
                CK(cudaFuncSetAttribute(k_bulk<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
                float ms = time_best([&] { k_bulk<1><<<148 * 4, 32, sm>>>(base, shadow, log, N / 16384, P, hdr, 16384, 3); });
                printf("bulk  1R+1W (log only), tile 16 KiB x 3, 4 CTA/SM                      %8.3f ms  %7.1f GB/s\n", ms, 2.0 * N / ms / 1e6);
            }
            if (hdr == 16) {
                struct C { u32 tile, stages, cps; };
                const C cv[] = {{16384, 3, 2}, {16384, 3, 3}, {8192, 4, 3}, {8192, 3, 4}, {4096, 4, 4}};
                for (const C& v : cv) {
                    if (v.tile > P) continue;
                    const size_t sm = ((sizeof(cc_crc_smem) + 127) / 128) * 128 + (size_t)v.tile * v.stages;
                    CK(cudaFuncSetAttribute(k_bulkcrc<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
                    float ms = time_best([&] { k_bulkcrc<8><<<148 * v.cps, 32 * 9, sm>>>(base, shadow, log, N / v.tile, P, hdr, v.tile, v.stages, d_tabs, crc_out); });
                    printf("bulk+crc 1R+2W, tile %2u KiB x %u, %u CTA/SM x (1+8) warps                %8.3f ms  %7.1f GB/s\n", v.tile >> 10, v.stages, v.cps, ms,
                           3.0 * N / ms / 1e6);
                    if (cudaGetLastError() != cudaSuccess) printf("   launch error\n");
                    check(P, hdr, "bulkcrc");
                }
                for (const C& v : cv) {
                    if (v.tile > P) continue;
                    const size_t sm = ((sizeof(cc_crc_smem) + 127) / 128) * 128 + (size_t)v.tile * v.stages;
                    CK(cudaFuncSetAttribute(k_bulkcrc<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
                    float ms = time_best([&] { k_bulkcrc<4><<<148 * v.cps, 32 * 5, sm>>>(base, shadow, log, N / v.tile, P, hdr, v.tile, v.stages, d_tabs, crc_out); });
                    printf("bulk+crc 1R+2W, tile %2u KiB x %u, %u CTA/SM x (1+4) warps                %8.3f ms  %7.1f GB/s\n", v.tile >> 10, v.stages, v.cps, ms,
                           3.0 * N / ms / 1e6);
                    check(P, hdr, "bulkcrc4");
                }
            }
        }
    }
    return 0;
}
