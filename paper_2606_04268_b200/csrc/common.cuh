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
constexpr uint32_t F_BLOCK_SUM = 1, F_SOURCE = 2, F_DEPTH = 4, F_PLACEHOLDER = 8, F_INDEX = 16;

// ---- tiling of the token stream: one tile = Params::tile consecutive sequences of one block.  The tile size belongs to
// the strategy: the bucketing kernel (k_pre: wave lists) sorts a tile's matches in shared memory and likes them large;
// the streaming kernels (k_pass, k_chain) want many small CTAs — measured on text1g_d4: PASSES 5.15 ms at 2048, 4.86 ms
// at 512; on fastq1g: k_pre 2.4 ms at 2048, 3.5 ms at 512; CHAIN 8.95 ms at 2048, 7.8 ms at 512.
constexpr int PRE_ITEMS = 8;                       // consecutive sequences per thread (8 x u16 = one 16 B load)
constexpr int PRE_THREADS = 256;                   // k_pre
constexpr int TILE_LIST = PRE_THREADS * PRE_ITEMS; // 2048: strategies LAUNCH / GRAPH / PERSISTENT
constexpr int PS_THREADS = 64;                     // k_pass
constexpr int TILE_STREAM = PS_THREADS * PRE_ITEMS;// 512: strategies PASSES / CHAIN
constexpr uint32_t PASS_MAX_DEPTH = 16;               // strategy PASSES: one streaming pass per depth, at most this many
constexpr uint32_t SMEM_DEPTHS = 4096;             // depth bins ranked in shared memory; deeper streams use global atomics

// ---- match kernel
#ifndef AX_PT
#define AX_PT 1024
#endif
constexpr int PERSIST_THREADS = AX_PT;             // k_waves: 1024 threads, one CTA per SM (measured best: DESIGN.md 6.2)
constexpr uint32_t SHORT_MAX = 32;                 // matches up to this length are copied by one thread
constexpr uint32_t LONG_LIT = 16;                  // literal runs longer than this are queued and copied by the whole grid (k_litcopy)
constexpr uint32_t LIT_PIECE = 4096;               // ... in pieces of at most this many bytes

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
    uint32_t n_final;                              // matches copied by the chain pass (checked against the header)
    uint32_t lit_q_count;                          // long literal runs queued for k_litcopy
    unsigned long long src_bytes_pre;              // M_src of the matches listed by the literal pass (strategy PASSES, sparse depths)
    uint32_t pad0[24];
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
    unsigned long long* tile_state;                // [n_tiles] exclusive (out << 32 | lit) prefix of the tile inside its block
    uint32_t* tile_blk;                            // [n_tiles] block index of the tile
    uint32_t* chain_sync;                          // strategy CHAIN: [32 + b] finished tiles of block b (complete only once blocks < b are)
    uint4* lit_q;                                  // [lit_q_cap] long literal runs: (dst, len, src offset in comp lo, hi)
    uint32_t lit_q_cap;
    uint32_t long_runs;                            // the header's mean literal run is 4-20 bytes (picks the literal pass instance)
    uint32_t* wl_dst;                              // [n_list] match destination (absolute)
    uint32_t* wl_off;                              // [n_list] match source (absolute)
    uint16_t* wl_len;                              // [n_list]
    uint64_t raw_size, comp_bytes;
    uint32_t block_size, n_blocks, n_tiles, tile, max_depth, min_match;   // tile: sequences per tile (TILE_LIST or TILE_STREAM)
    uint32_t n_list;                               // capacity of the wave lists = matches at depths 1 .. list_hi
    uint32_t list_hi;                              // depths 1 .. list_hi travel through wave lists (0: strategy CHAIN, no lists)
    uint32_t list_mask;                            // strategy PASSES: bit d set = depth d is sparse: the literal pass lists its
                                                   // matches and a list wave copies them; the other depths get a streaming pass
};

__host__ __device__ inline uint64_t pad16(uint64_t x) { return (x + 15) & ~(uint64_t)15; }

__device__ __forceinline__ void raise_fault(Status* st, uint32_t bits, uint32_t block) {
    atomicOr(&st->fault_flags, bits);
    atomicMin(&st->fault_block, block);
}

// ---- step a2, token parse: the 8 consecutive sequences of one thread from five 16-byte words (cmd, len, dep: 8 x u16;
// off: 8 x u32 in two words); entries at or past `n_valid` are zeroed (streams are padded to 16 bytes with zeros, but a
// tile's tail shares its last words with nothing — the mask is what makes them empty).
struct Seq8 { uint32_t c[PRE_ITEMS], l[PRE_ITEMS], dp[PRE_ITEMS], of[PRE_ITEMS]; };

__device__ __forceinline__ void unpack8(uint4 v, uint32_t (&x)[PRE_ITEMS]) {
    x[0] = v.x & 0xFFFFu; x[1] = v.x >> 16; x[2] = v.y & 0xFFFFu; x[3] = v.y >> 16;
    x[4] = v.z & 0xFFFFu; x[5] = v.z >> 16; x[6] = v.w & 0xFFFFu; x[7] = v.w >> 16;
}

__device__ __forceinline__ void parse8(Seq8& s, uint4 vc, uint4 vl, uint4 vd, uint4 o0, uint4 o1, uint32_t n_valid) {
    unpack8(vc, s.c); unpack8(vl, s.l); unpack8(vd, s.dp);
    s.of[0] = o0.x; s.of[1] = o0.y; s.of[2] = o0.z; s.of[3] = o0.w; s.of[4] = o1.x; s.of[5] = o1.y; s.of[6] = o1.z; s.of[7] = o1.w;
#pragma unroll
    for (int k = 0; k < PRE_ITEMS; ++k) if ((uint32_t)k >= n_valid) { s.c[k] = 0; s.l[k] = 0; s.dp[k] = 0; s.of[k] = 0; }
}

// The same from global memory: sequences j0 .. j0+7 of block B (j0 a multiple of 8).  need_src = false skips dep[] / off[].
__device__ __forceinline__ void load_seq8(Seq8& s, const uint8_t* comp, const BlockDesc& B, uint32_t j0, bool need_src) {
    const uint4 z = make_uint4(0u, 0u, 0u, 0u);
    if (j0 >= B.n_seq) { parse8(s, z, z, z, z, z, 0); return; }
    const uint4 vc = *reinterpret_cast<const uint4*>(comp + B.cmd_off + 2ull * j0);
    const uint4 vl = *reinterpret_cast<const uint4*>(comp + B.len_off + 2ull * j0);
    uint4 vd = z, o0 = z, o1 = z;
    if (need_src) {
        vd = *reinterpret_cast<const uint4*>(comp + B.dep_off + 2ull * j0);
        o0 = *reinterpret_cast<const uint4*>(comp + B.off_off + 4ull * j0);
        o1 = *reinterpret_cast<const uint4*>(comp + B.off_off + 4ull * j0 + 16);
    }
    parse8(s, vc, vl, vd, o0, o1, B.n_seq - j0);
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

// ---- cooperative copy of n bytes by a group of G lanes (gl = lane index inside the group), source and destination
// ranges disjoint.  dst: 16-byte aligned vector stores on the body, byte stores on head/tail; never stores outside
// [dst, dst+n).  src: whole aligned 16-byte words are loaded (plain L1-cached loads: callers order them after the
// producing wave by a kernel boundary or an acquiring grid barrier), so up to 15 bytes beyond either end of the source
// may be READ.  The body is unrolled by 4 so that four loads per lane are in flight (a long literal run or match is a
// memcpy: its rate is set by the loads in flight, not by the instruction count).
template <uint32_t G>
__device__ __forceinline__ void group_copy(uint8_t* dst, const uint8_t* src, uint32_t n, uint32_t gl) {
    uint32_t h = (uint32_t)(-(intptr_t)dst) & 15u;
    if (h > n) h = n;
    if (gl < h) dst[gl] = src[gl];
    if (G < 16 && gl + G < h) dst[gl + G] = src[gl + G];
    dst += h; src += h; n -= h;
    const uint32_t nvec = n >> 4;
    const uint32_t sh = (uint32_t)((uintptr_t)src & 15u);
    const uint4* s16 = reinterpret_cast<const uint4*>(src - sh);
    uint4* d16 = reinterpret_cast<uint4*>(dst);
    uint32_t v = gl;
    if (sh == 0) {
        for (; v + 3 * G < nvec; v += 4 * G) {
            const uint4 a = s16[v], b = s16[v + G], c = s16[v + 2 * G], d = s16[v + 3 * G];
            d16[v] = a; d16[v + G] = b; d16[v + 2 * G] = c; d16[v + 3 * G] = d;
        }
        for (; v < nvec; v += G) d16[v] = s16[v];
    } else {
        for (; v + 3 * G < nvec; v += 4 * G) {
            const uint4 a0 = s16[v], a1 = s16[v + 1], b0 = s16[v + G], b1 = s16[v + G + 1],
                        c0 = s16[v + 2 * G], c1 = s16[v + 2 * G + 1], e0 = s16[v + 3 * G], e1 = s16[v + 3 * G + 1];
            d16[v] = shift16(a0, a1, sh); d16[v + G] = shift16(b0, b1, sh);
            d16[v + 2 * G] = shift16(c0, c1, sh); d16[v + 3 * G] = shift16(e0, e1, sh);
        }
        for (; v < nvec; v += G) {
            const uint4 a = s16[v], b = s16[v + 1];
            d16[v] = shift16(a, b, sh);
        }
    }
    const uint32_t t = n & 15u, tb = nvec << 4;
    if (gl < t) dst[tb + gl] = src[tb + gl];
    if (G < 16 && gl + G < t) dst[tb + gl + G] = src[tb + gl + G];
}

__device__ __forceinline__ void warp_copy(uint8_t* dst, const uint8_t* src, uint32_t n, uint32_t lane) {
    group_copy<32>(dst, src, n, lane);
}

// ---- step a4, long literal runs: a run of more than LONG_LIT bytes is not copied by the thread that parsed it — one warp
// per run, run after run, leaves the warp waiting on one DRAM round trip per run, and a tile of incompressible data holds
// up to 2048 x 65 535 literal bytes (one CTA would copy 128 MB while the others idle): measured 7.7 ms of literal scatter
// on stress2g.  It is queued here, cut into pieces of at most LIT_PIECE bytes, and k_litcopy spreads the queue over the
// whole grid, eight lanes per piece.  Every piece is longer than LONG_LIT bytes, which bounds the queue by the
// header's total_lit.
// Warp-converged call; `has` selects the lanes that queue a run: one atomic per warp reserves the slots of all its lanes.
__device__ __forceinline__ void queue_long_literals(const Params& P, bool has, uint32_t dst, unsigned long long src_off, uint32_t len, uint32_t lane, uint32_t block) {
    if (!__any_sync(0xFFFFFFFFu, has)) return;
    const uint32_t np = has ? (len + LIT_PIECE - 1) / LIT_PIECE : 0u;
    uint32_t inc = np;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const uint32_t t = __shfl_up_sync(0xFFFFFFFFu, inc, d);
        if (lane >= (uint32_t)d) inc += t;
    }
    uint32_t base = 0;
    if (lane == 31) base = atomicAdd(&P.status->lit_q_count, inc);
    base = __shfl_sync(0xFFFFFFFFu, base, 31) + inc - np;
    if (np) {
        const uint32_t piece = (len + np - 1) / np;
        for (uint32_t k = 0, at = 0; k < np; ++k, at += piece) {
            const uint32_t n = len - at < piece ? len - at : piece;
            if (base + k < P.lit_q_cap) P.lit_q[base + k] = make_uint4(dst + at, n, (uint32_t)(src_off + at), (uint32_t)((src_off + at) >> 32));
            else raise_fault(P.status, F_BLOCK_SUM, block);  // more long runs than total_lit allows: the header lied
        }
    }
}

}  // namespace ax
