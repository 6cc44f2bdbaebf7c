// common.cuh — device-side data layout shared by the aceapex kernels (written from docs/FORMAT.md).
// Product code: shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace ax {

// ---- docs/FORMAT.md constants
constexpr uint32_t HDR_BYTES = 64, DIR_BYTES = 16, HIST_BYTES = 16;
constexpr uint32_t FLAG_FLATTENED = 1, FLAG_DEPTH_LIMITED = 2, FLAG_HAS_DEP = 4;

// ---- fault bits (include/aceapex.h ACEAPEX_F_*)
constexpr uint32_t F_BLOCK_SUM = 1, F_SOURCE = 2, F_DEPTH = 4, F_PLACEHOLDER = 8;

// ---- PRE kernel tiling: one tile = TILE consecutive sequences of one block
constexpr int PRE_THREADS = 256;
constexpr int PRE_ITEMS = 8;                       // consecutive sequences per thread (8 x u16 = one 16 B load)
constexpr int TILE = PRE_THREADS * PRE_ITEMS;      // 2048
constexpr uint32_t SMEM_DEPTHS = 4096;             // depth bins ranked in shared memory; deeper streams use global atomics

// ---- match kernel
#ifndef AX_PT
#define AX_PT 1024
#endif
constexpr int PERSIST_THREADS = AX_PT;             // k_waves: 1024 threads, one CTA per SM (measured best: DESIGN.md 6.2)
constexpr uint32_t SHORT_MAX = 32;
constexpr uint32_t FUSED_MAX_DEPTH = 16;           // the fused tile kernel handles streams up to this depth                 // matches up to this length are copied by one thread

// Per-block descriptor written by k_index (step a1).  Stream addresses are byte offsets from comp base.
struct BlockDesc {
    uint64_t cmd_off, len_off, dep_off, off_off, lit_off;
    uint64_t out_base;                             // b * block_size
    uint32_t n_seq, n_lit, raw_len, tile_base;     // tile_base = first global tile index of this block
};

// Status words at the start of scratch (one 256-byte slab; barrier counter on its own 128-byte line).
struct Status {
    uint32_t fault_flags;
    uint32_t fault_block;                          // atomicMin; 0xFFFFFFFF = none
    unsigned long long match_src_bytes;            // M_src counted during PRE
    uint32_t ticket;                               // dynamic tile counter of k_fused
    uint32_t n_match_seen;
    uint32_t pad0[26];
    uint32_t barrier;                              // grid barrier counter of the persistent wave kernel
    uint32_t pad1[31];
};
static_assert(sizeof(Status) == 256, "Status slab is 256 bytes");

// Everything a kernel needs, passed by value (fits the 4 KB parameter space easily).
struct Params {
    const uint8_t* comp;                           // device, compressed buffer
    uint8_t* out;                                  // device, decompressed output
    Status* status;
    uint32_t* wave_off;                            // [max_depth + 2]; wave d list = [wave_off[d], wave_off[d+1])
    uint32_t* cursor;                              // [max_depth + 2]; bucket cursors
    BlockDesc* blocks;                             // [n_blocks]
    unsigned long long* tile_state;                // [n_tiles] k_tilesum: exclusive (out << 32 | lit) prefix of the tile in its block
                                                   //           (k_fused: its decoupled look-back words)
    uint32_t* wl_dst;                              // [n_match] match destination (absolute)
    uint32_t* wl_off;                              // [n_match] match source (absolute)
    uint16_t* wl_len;                              // [n_match]
    uint32_t* prog;                                // [n_tiles] k_tilesum: block index of the tile (k_fused: phases completed per tile)
    uint32_t* front;                               // [FUSED_MAX_DEPTH + 2] fused kernel: leading tiles with prog >= p
    uint64_t raw_size;
    uint32_t block_size, n_blocks, n_tiles, max_depth, min_match, n_match;
};

__host__ __device__ inline uint64_t pad16(uint64_t x) { return (x + 15) & ~(uint64_t)15; }

__device__ __forceinline__ void raise_fault(Status* st, uint32_t bits, uint32_t block) {
    atomicOr(&st->fault_flags, bits);
    atomicMin(&st->fault_block, block);
}

// ---- 16-byte funnel shift: bytes [sh, sh+16) of the 32-byte value (a | b << 128), sh in 0..15
__device__ __forceinline__ uint4 shift16(uint4 a, uint4 b, uint32_t sh) {
    const uint32_t q = sh >> 2, r = (sh & 3) * 8;
    uint32_t w0, w1, w2, w3, w4;
    switch (q) {
        case 0: w0 = a.x; w1 = a.y; w2 = a.z; w3 = a.w; w4 = b.x; break;
        case 1: w0 = a.y; w1 = a.z; w2 = a.w; w3 = b.x; w4 = b.y; break;
        case 2: w0 = a.z; w1 = a.w; w2 = b.x; w3 = b.y; w4 = b.z; break;
        default: w0 = a.w; w1 = b.x; w2 = b.y; w3 = b.z; w4 = b.w; break;
    }
    uint4 o;
    o.x = __funnelshift_r(w0, w1, r);
    o.y = __funnelshift_r(w1, w2, r);
    o.z = __funnelshift_r(w2, w3, r);
    o.w = __funnelshift_r(w3, w4, r);
    return o;
}

// ---- warp-cooperative copy of n bytes, source and destination ranges disjoint.
// dst: 16-byte aligned vector stores on the body, byte stores on head/tail; never stores outside [dst, dst+n).
// src: whole aligned 16-byte words are loaded (plain L1-cached loads: callers order them after the producing wave
// by a kernel boundary or an acquiring grid barrier), so up to 15 bytes beyond either end of the source may be READ.
__device__ __forceinline__ void warp_copy(uint8_t* dst, const uint8_t* src, uint32_t n, uint32_t lane) {
    uint32_t h = (uint32_t)(-(intptr_t)dst) & 15u;
    if (h > n) h = n;
    if (lane < h) dst[lane] = src[lane];
    dst += h; src += h; n -= h;
    const uint32_t nvec = n >> 4;
    const uint32_t sh = (uint32_t)((uintptr_t)src & 15u);
    const uint4* s16 = reinterpret_cast<const uint4*>(src - sh);
    uint4* d16 = reinterpret_cast<uint4*>(dst);
    if (sh == 0) {
        for (uint32_t v = lane; v < nvec; v += 32) d16[v] = s16[v];
    } else {
        for (uint32_t v = lane; v < nvec; v += 32) {
            const uint4 a = s16[v], b = s16[v + 1];
            d16[v] = shift16(a, b, sh);
        }
    }
    const uint32_t t = n & 15u, tb = nvec << 4;
    if (lane < t) dst[tb + lane] = src[tb + lane];
}

}  // namespace ax
