// cc_crc.cuh -- CRC32C (Castagnoli, reflected 0x82F63B78) for the CUDA path.
//
// A GPU has no CRC instruction, so a page's CRC is assembled from independent pieces using
// the linearity of the CRC register over GF(2):
//   raw(M, init)      = register after feeding M starting from init (no final XOR)
//   raw(A||B, 0)      = raw(A, 0) * x^(8|B|)  XOR  raw(B, 0)          (mod G)
//   raw(M, ~0)        = raw(M, 0) XOR (~0) * x^(8|M|)
//   CRC32C(M)         = raw(M, ~0) XOR ~0
// A warp handles one 4 KiB segment: lane l owns the 16-byte vectors l, l+32, ..., l+224.  It
// runs the byte-table loop over each vector from 0 (8 independent chains -> ILP), folds them with
// Horner steps of x^(8*512), multiplies by its lane constant x^(8*16*(31-l)) (8 nibble-table
// lookups), the warp XORs the lanes together, and the warp multiplies by the segment constant
// x^(8*bytes after the segment) with one bit of the product per lane.
// The byte table and the nibble tables are replicated per lane in shared memory
// (entry*32 + lane) so the random lookups of the 32 lanes never collide on a bank.
#pragma once
#include "cc_common.cuh"

#define CC_CRC_POLY 0x82F63B78u

// ---- GF(2)[x] / G arithmetic in the reflected representation (bit 31 = x^0) ----
__host__ __device__ __forceinline__ u32 gf_mulx(u32 b) { return (b >> 1) ^ ((b & 1u) ? CC_CRC_POLY : 0u); }

__host__ __device__ inline u32 gf_mul(u32 a, u32 b) {
    u32 p = 0;
#pragma unroll 8
    for (int i = 0; i < 32; i++) {
        p ^= (a & (0x80000000u >> i)) ? b : 0u;
        b = gf_mulx(b);
    }
    return p;
}

// x^(8*nbytes) using the table xp[j] = x^(8*2^j)
__host__ __device__ inline u32 gf_xpow_bytes(const u32* xp, u64 nbytes) {
    u32 r = 0x80000000u;
    for (int j = 0; nbytes != 0 && j < 48; j++, nbytes >>= 1)
        if (nbytes & 1) r = gf_mul(r, xp[j]);
    return r;
}

// ---- host: build all constant tables ----
static inline void cc_crc_build_tables(cc_crc_tables* t) {
    for (u32 i = 0; i < 256; i++) {
        u32 c = i;
        for (int b = 0; b < 8; b++) c = gf_mulx(c);
        t->t0[i] = c;
    }
    for (int k = 1; k < 4; k++)                   // t0k[k-1][b]: byte b followed by k zero bytes (slicing-by-4)
        for (u32 i = 0; i < 256; i++) {
            const u32 prev = k == 1 ? t->t0[i] : t->t0k[k - 2][i];
            t->t0k[k - 1][i] = (prev >> 8) ^ t->t0[prev & 0xFFu];
        }
    u32 x8 = 0x80000000u;
    for (int b = 0; b < 8; b++) x8 = gf_mulx(x8);
    t->xp[0] = x8;
    for (int j = 1; j < 48; j++) t->xp[j] = gf_mul(t->xp[j - 1], t->xp[j - 1]);
    u32 s512 = gf_xpow_bytes(t->xp, 512);
    for (int b = 0; b < 4; b++)
        for (u32 v = 0; v < 256; v++) t->s512[b][v] = gf_mul(v << (8 * b), s512);
    for (u32 l = 0; l < 32; l++) t->lane_mul[l] = gf_xpow_bytes(t->xp, 16ull * (31 - l));
    for (u32 m = 0; m <= CC_SEG_POW_MAX; m++) t->seg_mul[m] = gf_xpow_bytes(t->xp, 4096ull * m);
    // lane_nib[(n*16 + v)*32 + l] = (v << 4n) * lane_mul[l]: multiply by the lane constant in 8 lookups
    for (u32 n = 0; n < 8; n++)
        for (u32 v = 0; v < 16; v++)
            for (u32 l = 0; l < 32; l++) t->lane_nib[(n * 16 + v) * 32 + l] = gf_mul(v << (4 * n), t->lane_mul[l]);
    // seg_pow[m*32 + i] = seg_mul[m] * x^i: multiply by the segment constant with one term per lane
    for (u32 m = 0; m <= CC_SEG_POW_MAX; m++) {
        u32 b = t->seg_mul[m];
        for (u32 i = 0; i < 32; i++) { t->seg_pow[m * 32 + i] = b; b = gf_mulx(b); }
    }
}

// ---- device: shared-memory tables ----
// t0 holds the byte table ROTATED LEFT BY 7 and replicated per lane: word (entry*32 + lane), i.e. byte
// offset entry*128 + lane*4.  The CRC register is kept rotated left by 7 as well ("z"), so the low
// byte of the register already sits at bits 7..14 = the table's byte offset: one LOP3 forms the
// address, one funnel shift + one LOP3 form the next state -> 3 ALU + 1 LDS per message byte.
struct alignas(16) cc_crc_smem {
    u32 t0[256 * 32];
    alignas(16) u32 lane_nib[8 * 16 * 32];
    alignas(16) u32 s512[4 * 256];
};

__device__ __forceinline__ u32 rotl32(u32 x, int n) { return __funnelshift_l(x, x, n); }
__device__ __forceinline__ u32 rotr32(u32 x, int n) { return __funnelshift_r(x, x, n); }

// Few, independent, coalesced global loads per thread (one latency, not a chain of them: the fill used to cost
// ~20 us of every launch): a warp loads 32 byte-table entries with ONE load and spreads them by shuffle; the
// other two tables are straight 16-byte copies.
__device__ __forceinline__ void cc_crc_smem_init(cc_crc_smem* s, const cc_crc_tables* g) {
    const u32 lane = threadIdx.x & 31u, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
    for (u32 e0 = w * 32u; e0 < 256u; e0 += nw * 32u) {
        const u32 mine = rotl32(g->t0[e0 + lane], 7);
#pragma unroll
        for (u32 e = 0; e < 32u; e++) s->t0[(e0 + e) * 32u + lane] = __shfl_sync(0xFFFFFFFFu, mine, e);
    }
    const uint4* nib = reinterpret_cast<const uint4*>(g->lane_nib);
    uint4* dn = reinterpret_cast<uint4*>(s->lane_nib);
    for (u32 i = threadIdx.x; i < 8 * 16 * 32 / 4; i += blockDim.x) dn[i] = nib[i];
    const uint4* s5 = reinterpret_cast<const uint4*>(&g->s512[0][0]);
    uint4* d5 = reinterpret_cast<uint4*>(s->s512);
    for (u32 i = threadIdx.x; i < 4 * 256 / 4; i += blockDim.x) d5[i] = s5[i];
    __syncthreads();
}

// z' for one message byte already XORed into z
__device__ __forceinline__ u32 crc_step_z(const char* t0, u32 lane4, u32 z) {
    const u32 v = *reinterpret_cast<const u32*>(t0 + ((z & 0x7F80u) | lane4));
    return v ^ (rotr32(z, 8) & 0x7FFFFF80u);
}

// raw register (init 0) over one 16-byte vector, memory order; returns the UNrotated register
__device__ __forceinline__ u32 crc_vec16(const cc_crc_smem* s, u32 lane4, const uint4& v) {
    const char* t0 = reinterpret_cast<const char*>(s->t0);
    const u32 w[4] = {v.x, v.y, v.z, v.w};
    u32 z = 0;
#pragma unroll
    for (int j = 0; j < 4; j++) {
        z ^= rotl32(w[j], 7);
#pragma unroll
        for (int b = 0; b < 4; b++) z = crc_step_z(t0, lane4, z);
    }
    return rotr32(z, 7);
}

// ---- slicing-by-4 variant (the applier's validation, which is bound by instruction issue) ----
// Four byte tables T3..T0 (byte followed by 3..0 zero bytes), each replicated per lane, laid out so that ONE byte-permute
// forms a lookup address: entry b of slice q sits at byte offset (q >> 1) * 65536 + b * 256 + (q & 1) * 128 + lane * 4 --
// PRMT(z, laneoff) puts byte k of the register into address bits 8..15 above the lane offset, no shift, no mask.
// A 32-bit step is 4 PRMT + 4 LDS + 2 LOP3 = 2.5 instructions per byte against 4.5 for the single table; 128 KiB of
// shared memory, so one 1,024-thread block per SM.
struct alignas(16) cc_crc_smem4 {
    u32 t[2 * 256 * 64];                    // 128 KiB
    alignas(16) u32 lane_nib[8 * 16 * 32];
    alignas(16) u32 s512[4 * 256];
};

__device__ __forceinline__ void cc_crc_smem_init(cc_crc_smem4* s, const cc_crc_tables* g) {
    const u32 lane = threadIdx.x & 31u, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
    // slice q uses table T(3-q): the FIRST message byte of a word is followed by three more
    for (u32 job = w; job < 4u * 8u; job += nw) {             // 4 slices x 8 groups of 32 entries
        const u32 q = job >> 3, e0 = (job & 7u) * 32u;
        const u32* src = q == 3 ? g->t0 : g->t0k[2 - q];
        const u32 mine = src[e0 + lane];
        u32* base = s->t + (q >> 1) * (256u * 64u) + (q & 1u) * 32u;
#pragma unroll
        for (u32 e = 0; e < 32u; e++) base[(e0 + e) * 64u + lane] = __shfl_sync(0xFFFFFFFFu, mine, e);
    }
    const uint4* nib = reinterpret_cast<const uint4*>(g->lane_nib);
    uint4* dn = reinterpret_cast<uint4*>(s->lane_nib);
    for (u32 i = threadIdx.x; i < 8 * 16 * 32 / 4; i += blockDim.x) dn[i] = nib[i];
    const uint4* s5 = reinterpret_cast<const uint4*>(&g->s512[0][0]);
    uint4* d5 = reinterpret_cast<uint4*>(s->s512);
    for (u32 i = threadIdx.x; i < 4 * 256 / 4; i += blockDim.x) d5[i] = s5[i];
    __syncthreads();
}

// one 32-bit step: the register after feeding the four bytes of z (already XORed with the message word)
__device__ __forceinline__ u32 crc_step32(const char* t, u32 lo, u32 hi, u32 z) {
    const u32 a0 = __byte_perm(z, lo, 0x5504), a1 = __byte_perm(z, hi, 0x5514);
    const u32 a2 = __byte_perm(z, lo, 0x5524), a3 = __byte_perm(z, hi, 0x5534);
    return *reinterpret_cast<const u32*>(t + a0) ^ *reinterpret_cast<const u32*>(t + a1) ^
           *reinterpret_cast<const u32*>(t + 65536 + a2) ^ *reinterpret_cast<const u32*>(t + 65536 + a3);
}
__device__ __forceinline__ u32 crc_vec16(const cc_crc_smem4* s, u32 lane4, const uint4& v) {
    const char* t = reinterpret_cast<const char*>(s->t);
    const u32 lo = lane4, hi = lane4 + 128u;
    u32 z = crc_step32(t, lo, hi, v.x);
    z = crc_step32(t, lo, hi, z ^ v.y);
    z = crc_step32(t, lo, hi, z ^ v.z);
    return crc_step32(t, lo, hi, z ^ v.w);
}

__device__ __forceinline__ u32 crc_shift512(const u32* s512, u32 v) {
    return s512[v & 0xFFu] ^ s512[256 + ((v >> 8) & 0xFFu)] ^ s512[512 + ((v >> 16) & 0xFFu)] ^ s512[768 + (v >> 24)];
}

// acc * lane_mul[lane] through the lane-replicated nibble tables (conflict-free, 8 lookups)
__device__ __forceinline__ u32 crc_lane_mul(const u32* lane_nib, u32 lane4, u32 acc) {
    const char* nb = reinterpret_cast<const char*>(lane_nib);
    u32 r = 0;
#pragma unroll
    for (int n = 0; n < 8; n++) {
        const u32 sh = (n * 4 >= 7) ? (acc >> (n * 4 - 7)) : (acc << (7 - n * 4));
        r ^= *reinterpret_cast<const u32*>(nb + n * 2048 + ((sh & 0x780u) | lane4));
    }
    return r;
}

// Warp-level raw CRC contribution of one segment of nv (<= 256) 16-byte vectors held as
// v[u] = vector (lane + 32u); `after` = bytes of the message that follow this segment.
// Returns (in every lane) raw(segment, 0) * x^(8*after).
// SM: the shared-memory table set (cc_crc_smem: one byte table, 4 instructions per byte; cc_crc_smem4: slicing-by-4).
template <int U, class SM>
__device__ __forceinline__ u32 crc_segment_warp(const SM* s, const cc_crc_tables* g, const uint4 (&v)[U],
                                                u32 nv, u64 after, u32 lane) {
    const u32 lane4 = lane << 2;
    u32 acc = 0;
    if (nv == 32u * U) {
        u32 part[U];
#pragma unroll
        for (int u = 0; u < U; u++) part[u] = crc_vec16(s, lane4, v[u]);      // U independent chains
#pragma unroll
        for (int u = 0; u < U; u++) acc = (u ? crc_shift512(s->s512, acc) : 0u) ^ part[u];
        acc = crc_lane_mul(s->lane_nib, lane4, acc);
    } else {
        int last = -1;
#pragma unroll
        for (int u = 0; u < U; u++) {
            if (lane + 32u * u < nv) {
                acc = crc_shift512(s->s512, acc) ^ crc_vec16(s, lane4, v[u]);
                last = u;
            }
        }
        if (last >= 0) {
            u32 j_last = lane + 32u * (u32)last;
            acc = gf_mul(acc, gf_xpow_bytes(g->xp, 16ull * (nv - 1 - j_last)));
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc ^= __shfl_xor_sync(0xFFFFFFFFu, acc, o);
    if (after != 0) {
        if ((after & 4095u) == 0 && (after >> 12) <= CC_SEG_POW_MAX) {
            // acc * seg_mul[m]: lane i contributes bit (31-i) of acc times seg_mul[m]*x^i
            u32 term = ((acc >> (31 - lane)) & 1u) ? g->seg_pow[(u32)(after >> 12) * 32 + lane] : 0u;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) term ^= __shfl_xor_sync(0xFFFFFFFFu, term, o);
            acc = term;
        } else {
            acc = gf_mul(acc, gf_xpow_bytes(g->xp, after));
        }
    }
    return acc;
}

// Finalise: XOR of all segment contributions -> CRC32C.  init_term = 0xFFFFFFFF * x^(8*len), which
// is precomputed per region for its full and its tail page length.
__device__ __forceinline__ u32 crc_finalize(u32 acc, u32 init_term) { return acc ^ init_term ^ 0xFFFFFFFFu; }

// Serial CRC32C of a few bytes (commit payload), single thread: bit by bit in registers -- 128 shift/xor steps
// for a commit payload, cheaper than 16 dependent lookups in a global table that is cold in this SM's L1.
__device__ inline u32 crc_serial(const cc_crc_tables*, const u8* p, u32 n) {
    u32 c = 0xFFFFFFFFu;
    for (u32 i = 0; i < n; i++) {
        c ^= p[i];
#pragma unroll
        for (int b = 0; b < 8; b++) c = gf_mulx(c);
    }
    return c ^ 0xFFFFFFFFu;
}

// Combine one segment's CRC contribution into its record's 64-bit state word and tell whether this
// was the record's last segment.  For nseg <= 32 a single 64-bit atomicXor carries both the
// contribution (low half) and the segment's done bit (high half), so no fence is needed: the
// thread that sees every other bit already set is the finisher and the returned old value holds
// the XOR of all other contributions.  Longer records fall back to XOR + fence + counter.
// Returns true for the finisher, with *acc = XOR of all contributions; the state word is left zero.
// Segments c0 .. c0 + cn - 1 at once (contrib = XOR of their contributions).
__device__ __forceinline__ bool crc_record_combine_n(u64* state, u32 nseg, u32 c0, u32 cn, u32 contrib, u32* acc) {
    if (cn == nseg) { *acc = contrib; return true; }
    if (nseg <= 32) {
        const u32 full = nseg == 32 ? 0xFFFFFFFFu : ((1u << nseg) - 1u);
        const u32 mine = (cn == 32 ? 0xFFFFFFFFu : ((1u << cn) - 1u)) << c0;
        const u64 old = atomicXor(reinterpret_cast<unsigned long long*>(state), ((u64)mine << 32) | contrib);
        if (((u32)(old >> 32) | mine) != full) return false;
        *acc = (u32)old ^ contrib;
        *state = 0;
        return true;
    }
    atomicXor(reinterpret_cast<unsigned long long*>(state), (u64)contrib);
    __threadfence();
    const u64 old = atomicAdd(reinterpret_cast<unsigned long long*>(state), (u64)cn << 32);
    if ((u32)(old >> 32) != nseg - cn) return false;
    __threadfence();
    *acc = (u32)atomicExch(reinterpret_cast<unsigned long long*>(state), 0ull);
    return true;
}
__device__ __forceinline__ bool crc_record_combine(u64* state, u32 nseg, u32 c, u32 contrib, u32* acc) {
    return crc_record_combine_n(state, nseg, c, 1u, contrib, acc);
}
