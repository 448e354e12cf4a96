// cc_static.cu -- cc_dirty_pages_static: the dirty scan + ordered compaction (steps a1-a2)
// for callers that must not allocate.  A translation unit of its own: nothing in concordia.cu changes.
//
// Who needs this.  The regular path keeps its scratch (dirty bitmap, tickets, look-back words) in a workspace
// the caller allocates per region, and a context (cc_init) that allocates control blocks.  Three kinds of
// caller cannot do either at the moment they want a dirty list:
//   * code that runs next to a resident persistent kernel -- the paper's own setting: cudaMalloc and
//     cudaFree synchronise the device and can wait forever on a kernel that never exits;
//   * an inference server that handed all of HBM to its KV-cache pool at start-up: a later cudaMalloc simply
//     fails, and the pool's allocator is not ours to call;
//   * a fault handler or watchdog that wants to know what changed since the last commit BEFORE it decides
//     anything, and must not disturb the allocator state it is about to inspect.
// For them the scratch lives in the library image: one file-scope __device__ array, sized for
// CC_STATIC_MAX_PAGES pages (2 MiB + 256 B).  Every GPU that loads libconcordia.so carries it until the
// process exits, whether or not this call is ever made.
//
// The kernel is cc_scan_kernel's compare loop (cc_scan_items, shared source) followed, in the same launch, by
// an in-order ranking of the bitmap by whichever block finishes last -- no second launch, no look-back words,
// no assumption that the grid is co-resident.
#include <cstdint>
#include <cstring>
#include <mutex>

#include "cc_common.cuh"
#include "cc_ckpt.cuh"

#define CC_STATIC_CTL_BYTES 256u
#define CC_STATIC_BITMAP_BYTES (CC_STATIC_MAX_PAGES / 8u)
#define CC_STATIC_SCRATCH_BYTES (CC_STATIC_CTL_BYTES + CC_STATIC_BITMAP_BYTES)
#define CC_STATIC_THREADS 256
#define CC_STATIC_MAX_DEVICES 64

static_assert(CC_STATIC_MAX_PAGES % (32u * CC_COMPACT_TILE_WORDS) == 0, "the bitmap is a whole number of ranking tiles");
static_assert(CC_STATIC_THREADS == CC_COMPACT_THREADS, "one uint4 of bitmap words per thread and tile");

// [0, 256): control words.  [256, end): one bit per page.  In HOST code this name is only a handle for
// cudaGetSymbolAddress -- it is not a device address and must never be handed to a kernel as one.
static __device__ __align__(256) unsigned char cc_static_scratch[CC_STATIC_SCRATCH_BYTES];

struct cc_static_ctl {
    u32 blocks_done;        // blocks that have finished their share of the compare
    u32 pad[63];
};
static_assert(sizeof(cc_static_ctl) == CC_STATIC_CTL_BYTES, "control block is 256 bytes");

__global__ void __launch_bounds__(CC_STATIC_THREADS) cc_dirty_pages_static_kernel(const __grid_constant__ cc_region_dev rg, cc_static_ctl* ctl,
                                                                                  u32* d_list, u32 list_capacity, u32* d_count) {
    __shared__ u32 s_last;
    __shared__ u32 s_warp[CC_STATIC_THREADS / 32];
    const u32 tid = threadIdx.x, lane = tid & 31u, wid = tid >> 5;

    // a1: every warp compares its pages and sets their bits (bitmap all zero on entry: the host call cleared it)
    const cc_grid g = cc_hw_grid();
    cc_scan_items<8>(rg, g.warp(), g.nwarps());

    // the block that counts out last has every other block's bits behind its fence
    __threadfence();
    __syncthreads();
    if (tid == 0) s_last = (atomicAdd(&ctl->blocks_done, 1u) == gridDim.x - 1) ? 1u : 0u;
    __syncthreads();
    if (!s_last) return;
    __threadfence();

    // a2: ascending list of the set bits, tile by tile in order; `base` = dirty pages before this tile
    const u32 nt = (u32)((rg.n_words + CC_COMPACT_TILE_WORDS - 1) / CC_COMPACT_TILE_WORDS);
    u32 base = 0;
    for (u32 t = 0; t < nt; t++) {
        const u64 w0 = (u64)t * CC_COMPACT_TILE_WORDS + (u64)tid * 4u;
        const uint4 q = __ldcg(reinterpret_cast<const uint4*>(&rg.bitmap[w0]));
        const u32 cnt = __popc(q.x) + __popc(q.y) + __popc(q.z) + __popc(q.w);
        if (!__syncthreads_or(cnt != 0)) continue;              // a clean tile (the usual case) costs one load
        u32 inc = cnt;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const u32 n = __shfl_up_sync(0xFFFFFFFFu, inc, o);
            if (lane >= o) inc += n;
        }
        if (lane == 31) s_warp[wid] = inc;
        __syncthreads();
        u32 warp_base = 0, total = 0;
        for (u32 i = 0; i < CC_STATIC_THREADS / 32; i++) {
            const u32 v = s_warp[i];
            if (i < wid) warp_base += v;
            total += v;
        }
        u32 pos = base + warp_base + (inc - cnt);
        const u32 wv[4] = {q.x, q.y, q.z, q.w};
#pragma unroll
        for (u32 i = 0; i < 4; i++) {
            u32 w = wv[i];
            const u64 pbase = (w0 + i) << 5;
            while (w) {
                const u32 bit = __ffs(w) - 1;
                w &= w - 1;
                if (pos < list_capacity) d_list[pos] = (u32)(pbase + bit);
                pos++;
            }
        }
        base += total;
        __syncthreads();                                        // s_warp is reused by the next dirty tile
    }
    if (tid == 0) *d_count = base;
}

// ---------------------------------------------------------------------------------------- host side --

struct cc_static_device {
    int state;              // 0 = not set up (a failed set-up is tried again by the next call), 1 = ready
    unsigned char* scratch; // DEVICE address of cc_static_scratch on this GPU
    int sm_count;
    int blocks_per_sm;
};
static cc_static_device g_static_dev[CC_STATIC_MAX_DEVICES];
static std::mutex g_static_mu;

// Once per device, with that device current: resolve the array's device address and the launch geometry.
// No allocation of ours; the runtime may load this module's code onto the GPU here, which is why the first
// call on a device belongs before any stream capture.
static cudaError_t cc_static_setup(int device, cc_static_device** out) {
    std::lock_guard<std::mutex> lk(g_static_mu);
    cc_static_device* d = &g_static_dev[device];
    if (d->state == 0) {
        void* p = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&p, cc_static_scratch);
        if (e == cudaSuccess) e = cudaDeviceGetAttribute(&d->sm_count, cudaDevAttrMultiProcessorCount, device);
        if (e == cudaSuccess)
            e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&d->blocks_per_sm, cc_dirty_pages_static_kernel, CC_STATIC_THREADS, 0);
        if (e == cudaSuccess && (p == nullptr || d->sm_count <= 0 || d->blocks_per_sm <= 0)) e = cudaErrorInvalidValue;
        if (e != cudaSuccess) {
            (void)cudaGetLastError();
            return e;
        }
        d->scratch = static_cast<unsigned char*>(p);
        d->state = 1;
    }
    *out = d;
    return cudaSuccess;
}

extern "C" int32_t cc_dirty_pages_static(int32_t device, const void* cur, const void* shadow, uint64_t bytes, uint32_t page_bytes,
                                         uint32_t* d_list, uint32_t list_capacity, uint32_t* d_count, void* stream,
                                         int32_t* cuda_error) {
    if (cuda_error) *cuda_error = 0;
    if (device < 0 || device >= CC_STATIC_MAX_DEVICES) return CC_ERR_INVALID;
    if (!cur || !shadow || !d_count || (list_capacity && !d_list)) return CC_ERR_INVALID;
    if (((uintptr_t)cur & 15u) || ((uintptr_t)shadow & 15u) || ((uintptr_t)d_list & 3u) || ((uintptr_t)d_count & 3u)) return CC_ERR_INVALID;
    if (page_bytes == 0 || (page_bytes & 15u) || bytes == 0 || (bytes & 15ull)) return CC_ERR_INVALID;
    const uint64_t n_pages = (bytes + page_bytes - 1) / page_bytes;
    if (n_pages > CC_STATIC_MAX_PAGES) return CC_ERR_STATIC_LIMIT;      // the built-in bitmap has one bit per page and no more

    int prev = -1;
    cudaError_t e = cudaGetDevice(&prev);
    if (e == cudaSuccess && prev != device) e = cudaSetDevice(device);
    cc_static_device* d = nullptr;
    if (e == cudaSuccess) e = cc_static_setup(device, &d);
    if (e == cudaSuccess) {
        cc_region_dev r;
        memset(&r, 0, sizeof(r));
        r.base = (u8*)cur;
        r.shadow = (u8*)shadow;
        r.bytes = bytes;
        r.n_pages = n_pages;
        r.page_bytes = page_bytes;
        r.spp = (page_bytes + CC_SEG_BYTES - 1) / CC_SEG_BYTES;
        r.n_words = (n_pages + 31) / 32;
        r.bitmap = reinterpret_cast<u32*>(d->scratch + CC_STATIC_CTL_BYTES);
        const uint64_t n_tiles = (r.n_words + CC_COMPACT_TILE_WORDS - 1) / CC_COMPACT_TILE_WORDS;
        const cudaStream_t st = (cudaStream_t)stream;
        // the array still holds whatever the previous call (or a call that died half-way) left: the counter and the
        // part of the bitmap this call reads start at zero
        e = cudaMemsetAsync(d->scratch, 0, CC_STATIC_CTL_BYTES + n_tiles * CC_COMPACT_TILE_WORDS * 4ull, st);
        if (e == cudaSuccess) {
            const uint64_t wpb = CC_STATIC_THREADS / 32;
            uint64_t grid = (n_pages * (uint64_t)r.spp + wpb - 1) / wpb;
            const uint64_t cap = (uint64_t)d->sm_count * (uint64_t)d->blocks_per_sm;
            if (grid > cap) grid = cap;
            cc_dirty_pages_static_kernel<<<(unsigned)grid, CC_STATIC_THREADS, 0, st>>>(
                r, reinterpret_cast<cc_static_ctl*>(d->scratch), d_list, list_capacity, d_count);
            e = cudaGetLastError();
        }
    }
    if (prev >= 0 && prev != device) (void)cudaSetDevice(prev);
    if (e != cudaSuccess) {
        if (cuda_error) *cuda_error = (int32_t)e;
        return CC_ERR_CUDA;
    }
    return CC_OK;
}
