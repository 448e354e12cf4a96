// cc_fused.cuh -- building blocks of the single-pass checkpoint (cc_pass.cuh): the warp-wide decoupled look-back over
// tile status words, and the warp-cooperative multiply of a CRC register by x^(8*4096).
#pragma once
#include "cc_common.cuh"
#include "cc_crc.cuh"
#include "cc_ckpt.cuh"

// Warp-wide decoupled look-back: sum of the dirty counts of tiles [0, t).  The status words are read and
// written with RELAXED gpu-scope accesses: the count a word carries is the whole message (nothing else a tile
// wrote is read by another tile inside this kernel), and a release here would make the publishing warp wait
// for its earlier record stores -- over the host link with a pinned log -- and stall every tile behind it.  blocking = false gives up
// (returns false) as soon as a predecessor that has not published yet is met before an inclusive one, or after max_steps
// groups of 32 aggregates.
__device__ __forceinline__ bool cc_fused_lookback(const u64* status, u32 run, u32 t, u32 lane, bool blocking, u32* excl_out,
                                                  u32 max_steps = 0xFFFFFFFFu) {
    u32 excl = 0;
    int base = (int)t - 1;
    for (u32 step = 0;; step++) {
        if (!blocking && step >= max_steps) return false;
        const int j = base - (int)lane;
        u64 s = lb_pack(run, CC_LB_INC, 0);                 // virtual tile -1: inclusive sum 0
        if (j >= 0) s = ld_relaxed_gpu_u64(&status[j]);
        const u32 flag = (u32)(s >> 32) & 3u;
        const bool valid = ((u32)(s >> 34) == run) && flag != 0;
        const u32 inv = __ballot_sync(0xFFFFFFFFu, !valid);
        const u32 inc = __ballot_sync(0xFFFFFFFFu, valid && flag == (u32)CC_LB_INC);
        const u32 first_inv = inv ? (u32)__ffs(inv) - 1u : 32u;
        const u32 first_inc = inc ? (u32)__ffs(inc) - 1u : 32u;
        if (first_inc < first_inv) {                        // nearest inclusive predecessor, all nearer ones valid
            excl += __reduce_add_sync(0xFFFFFFFFu, lane <= first_inc ? (u32)s : 0u);
            *excl_out = excl;
            return true;
        }
        if (first_inv < 32u) {                              // someone has not published yet
            if (!blocking) return false;
            __nanosleep(40);
            continue;
        }
        excl += __reduce_add_sync(0xFFFFFFFFu, (u32)s);     // 32 aggregates: keep walking
        base -= 32;
    }
}

// acc * x^(8*4096): lane i contributes bit (31-i) of acc times pow_lane = x^(8*4096) * x^i.
__device__ __forceinline__ u32 cc_warp_mul_seg(u32 acc, u32 pow_lane, u32 lane) {
    u32 term = ((acc >> (31 - lane)) & 1u) ? pow_lane : 0u;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) term ^= __shfl_xor_sync(0xFFFFFFFFu, term, o);
    return term;
}

