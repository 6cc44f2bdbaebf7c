// k_fused.cu — steps a2-a7 in ONE kernel for shallow streams (max_depth <= FUSED_MAX_DEPTH, e.g. the depth-limited
// encoder of PAPER.md:228 §7.4): token parse, segmented scan, literal scatter and all match waves, tile by tile,
// with the tile's OUTPUT assembled in shared memory.
//
// Why: matches average 5-9 bytes, so a wave that writes them straight to global
// memory issues ~3 sub-word stores per match; measured on B200 the L2 sustains only ~30 G matches/s of that
// (one 8-byte gather + three small scattered stores per item), against 244 G/s for gathers alone.  Here the small
// stores land in shared memory and the tile leaves the SM as whole 16-byte coalesced words; no wave lists are
// written or read (20 bytes per match saved) and the compressed stream is read exactly once.
//
// Order (a7) without a grid barrier: a tile = TILE consecutive sequences of one block; CTAs take tiles in file
// order from a ticket counter and keep a tile through phases p = 0 (literals), 1 .. max_depth (matches of depth p).
// After each phase the tile's span is flushed to `out` and prog[tile] = p + 1 is published (release).  Phase p of
// tile T starts when every tile T' < T has prog >= p: a depth-p match reads bytes of depth <= p-1,
// all of them in tiles <= T because off < mdst.  front[p] caches the number of leading tiles known to satisfy that.
// Tiles are claimed in order, so a waiting tile only ever waits for tiles held by resident CTAs: no deadlock.
#include "common.cuh"
#include "copy.cuh"

namespace ax {

constexpr unsigned long long FST_AGG = 1ull << 62, FST_INC = 2ull << 62, FST_MASK = 3ull << 62;
constexpr uint32_t FSAT = 0x3FFFFFFFu;
constexpr uint32_t OB_BYTES = 40 * 1024;             // shared-memory image of the tile's output span

__device__ __forceinline__ unsigned long long f_pack(unsigned long long flag, uint32_t so, uint32_t sl) {
    so = so > FSAT ? FSAT : so; sl = sl > FSAT ? FSAT : sl;
    return flag | ((unsigned long long)so << 31) | (unsigned long long)sl;
}
__device__ __forceinline__ unsigned long long f_ld64(const unsigned long long* p) {
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void f_st64(unsigned long long* p, unsigned long long v) {
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ uint32_t f_ld32(const uint32_t* p) {
    uint32_t v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

struct FusedSmem {
    unsigned long long warp_sum[PRE_THREADS / 32];
    unsigned long long tile_prefix;                  // (out << 32) | lit of everything before this tile in its block
    unsigned long long tile_total;
    unsigned long long depth_mask;                   // bit d: the tile has a match of depth d (d <= 63)
    uint32_t tile;
    uint32_t cnt[FUSED_MAX_DEPTH + 3];               // matches per depth in this tile (checked against the header histogram)
    uint32_t dstart[FUSED_MAX_DEPTH + 3];            // depth-sorted entry list: depth d occupies [dstart[d], dstart[d+1])
    uint16_t wcnt[PRE_THREADS / 32][FUSED_MAX_DEPTH + 2];   // per warp, per depth: matches, then exclusive base in the list
    uint32_t e_dst[TILE];                            // the tile's matches sorted by depth
    uint32_t e_off[TILE];
    uint16_t e_len[TILE];
    __align__(16) uint8_t ob[OB_BYTES + 32];
};

// Publish "phases < p done" for this tile: every thread's stores (the flush) happen-before the release store.
__device__ __forceinline__ void publish(uint32_t* prog, uint32_t tile, uint32_t p) {
    __syncthreads();
    if (threadIdx.x == 0) asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(prog + tile), "r"(p) : "memory");
}

// Wait until every tile < `tile` has prog >= p.  Warp 0 advances the shared frontier front[p]; the final acquire
// fence also invalidates L1 (CCTL.IVALL), so the plain loads that follow see what other SMs flushed.
__device__ __forceinline__ void wait_ready(const Params& P, uint32_t tile, uint32_t p) {
    if (tile != 0 && threadIdx.x < 32) {
        const uint32_t lane = threadIdx.x;
        uint32_t f = 0;
        if (lane == 0) f = f_ld32(P.front + p);
        f = __shfl_sync(0xFFFFFFFFu, f, 0);
        const uint32_t f0 = f;
        while (f < tile) {
            // 128 flags per round trip (4 per lane); lead = number of leading flags that are >= p
            uint32_t v[4];
#pragma unroll
            for (int r = 0; r < 4; ++r) { const uint32_t idx = f + 32u * r + lane; v[r] = idx < tile ? f_ld32(P.prog + idx) : 0xFFFFFFFFu; }
            uint32_t lead = 0;
#pragma unroll
            for (int r = 0; r < 4; ++r) {
                const uint32_t notok = __ballot_sync(0xFFFFFFFFu, v[r] < p);
                if (lead == 32u * r) lead += notok ? (uint32_t)__ffs(notok) - 1u : 32u;
            }
            f = f + lead < tile ? f + lead : tile;
            if (lead == 0) __nanosleep(32);
        }
        if (lane == 0) {
            asm volatile("fence.acq_rel.gpu;" ::: "memory");
            if (f > f0) atomicMax(P.front + p, f);
        }
    }
    __syncthreads();
}

// Copy the tile image [t0, t1) from shared memory to out: byte stores up to the first 16-byte boundary and after
// the last one (neighbouring bytes belong to other tiles), 16-byte coalesced stores in between.
__device__ __forceinline__ void flush_tile(uint8_t* out, const uint8_t* img, uint32_t t0, uint32_t t1) {
    // img + x addresses byte x of the output (img is pre-biased; img + (t0 & ~15) is 16-byte aligned)
    const uint32_t a0 = (t0 + 15u) & ~15u, a1 = t1 & ~15u;
    if (a0 >= a1) { for (uint32_t x = t0 + threadIdx.x; x < t1; x += PRE_THREADS) out[x] = img[x]; return; }
    if (threadIdx.x < a0 - t0) out[t0 + threadIdx.x] = img[t0 + threadIdx.x];
    if (threadIdx.x < t1 - a1) out[a1 + threadIdx.x] = img[a1 + threadIdx.x];
    const uint4* s = reinterpret_cast<const uint4*>(img + a0);
    uint4* d = reinterpret_cast<uint4*>(out + a0);
    const uint32_t nv = (a1 - a0) >> 4;
    for (uint32_t v = threadIdx.x; v < nv; v += PRE_THREADS) d[v] = s[v];
}

__global__ void __launch_bounds__(PRE_THREADS, 3) k_fused(Params P) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    FusedSmem& S = *reinterpret_cast<FusedSmem*>(smem_raw);
    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    unsigned long long src_bytes = 0;

    for (;;) {
        __syncthreads();
        if (tid == 0) { S.tile = atomicAdd(&P.status->ticket, 1u); S.depth_mask = 0ull; }
        if (tid <= FUSED_MAX_DEPTH) S.cnt[tid] = 0;
        __syncthreads();
        const uint32_t tile = S.tile;
        if (tile >= P.n_tiles) break;
        // ---- which block: last b with tile_base[b] <= tile
        uint32_t lo = 0, hi = P.n_blocks - 1;
        while (lo < hi) {
            const uint32_t mid = (lo + hi + 1) >> 1;
            if (P.blocks[mid].tile_base <= tile) lo = mid; else hi = mid - 1;
        }
        const uint32_t b = lo;
        const BlockDesc B = P.blocks[b];
        const uint32_t t_in_blk = tile - B.tile_base;
        const uint32_t j0 = t_in_blk * TILE + tid * PRE_ITEMS;
        // ---- a2: parse
        uint32_t c[PRE_ITEMS], l[PRE_ITEMS], dp[PRE_ITEMS], of[PRE_ITEMS];
        if (j0 < B.n_seq) {
            const uint4 vc = *reinterpret_cast<const uint4*>(P.comp + B.cmd_off + 2ull * j0);
            const uint4 vl = *reinterpret_cast<const uint4*>(P.comp + B.len_off + 2ull * j0);
            const uint4 vd = *reinterpret_cast<const uint4*>(P.comp + B.dep_off + 2ull * j0);
            const uint4 o0 = *reinterpret_cast<const uint4*>(P.comp + B.off_off + 4ull * j0);
            const uint4 o1 = *reinterpret_cast<const uint4*>(P.comp + B.off_off + 4ull * j0 + 16);
            const uint32_t wc[4] = {vc.x, vc.y, vc.z, vc.w}, wl[4] = {vl.x, vl.y, vl.z, vl.w}, wd[4] = {vd.x, vd.y, vd.z, vd.w};
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                c[2 * k] = wc[k] & 0xFFFFu; c[2 * k + 1] = wc[k] >> 16;
                l[2 * k] = wl[k] & 0xFFFFu; l[2 * k + 1] = wl[k] >> 16;
                dp[2 * k] = wd[k] & 0xFFFFu; dp[2 * k + 1] = wd[k] >> 16;
            }
            of[0] = o0.x; of[1] = o0.y; of[2] = o0.z; of[3] = o0.w; of[4] = o1.x; of[5] = o1.y; of[6] = o1.z; of[7] = o1.w;
#pragma unroll
            for (int k = 0; k < PRE_ITEMS; ++k) if (j0 + k >= B.n_seq) { c[k] = 0; l[k] = 0; dp[k] = 0; of[k] = 0; }
        } else {
#pragma unroll
            for (int k = 0; k < PRE_ITEMS; ++k) { c[k] = 0; l[k] = 0; dp[k] = 0; of[k] = 0; }
        }
        // ---- a3: scan of (cmd+len, cmd) packed as (hi, lo) of one u64
        unsigned long long tsum = 0;
#pragma unroll
        for (int k = 0; k < PRE_ITEMS; ++k) tsum += ((unsigned long long)(c[k] + l[k]) << 32) | c[k];
        unsigned long long inc = tsum;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const unsigned long long t = __shfl_up_sync(0xFFFFFFFFu, inc, d);
            if (lane >= d) inc += t;
        }
        if (lane == 31) S.warp_sum[warp] = inc;
        __syncthreads();
        unsigned long long wpre = 0, total = 0;
#pragma unroll
        for (int w = 0; w < PRE_THREADS / 32; ++w) {
            const unsigned long long x = S.warp_sum[w];
            if (w < (int)warp) wpre += x;
            total += x;
        }
        if (tid == 0) {   // decoupled look-back along this block's tiles
            const uint32_t tot_o = (uint32_t)(total >> 32), tot_l = (uint32_t)total;
            uint32_t pre_o = 0, pre_l = 0;
            if (t_in_blk != 0) {
                f_st64(&P.tile_state[tile], f_pack(FST_AGG, tot_o, tot_l));
                uint32_t q = tile;
                for (;;) {
                    --q;
                    unsigned long long s;
                    do { s = f_ld64(&P.tile_state[q]); } while ((s & FST_MASK) == 0);
                    pre_o += (uint32_t)((s >> 31) & 0x7FFFFFFFu); pre_l += (uint32_t)(s & 0x7FFFFFFFu);
                    if (pre_o > FSAT) pre_o = FSAT;
                    if (pre_l > FSAT) pre_l = FSAT;
                    if ((s & FST_MASK) == FST_INC) break;
                }
            }
            f_st64(&P.tile_state[tile], f_pack(FST_INC, pre_o + tot_o, pre_l + tot_l));
            S.tile_prefix = ((unsigned long long)pre_o << 32) | pre_l;
            S.tile_total = total;
            const bool last_tile = (t_in_blk + 1) * (uint32_t)TILE >= B.n_seq;
            if (last_tile && (pre_o + tot_o != B.raw_len || pre_l + tot_l != B.n_lit)) raise_fault(P.status, F_BLOCK_SUM, b);
        }
        __syncthreads();
        const unsigned long long ex = S.tile_prefix + wpre + (inc - tsum);
        uint32_t pos = (uint32_t)(ex >> 32);                 // output offset inside the block
        uint32_t lsrc = (uint32_t)ex;                        // offset inside the block's lit[]
        // ---- the tile's output span [t0, t1) (absolute, clamped to the block so a corrupt stream stays in bounds)
        const uint32_t blk_lo = (uint32_t)B.out_base, blk_hi = blk_lo + B.raw_len;
        uint32_t t0 = blk_lo + (uint32_t)(S.tile_prefix >> 32), t1 = t0 + (uint32_t)(S.tile_total >> 32);
        if (t0 > blk_hi) t0 = blk_hi;
        if (t1 > blk_hi || t1 < t0) t1 = blk_hi;
        const uint32_t tb = t0 & ~15u;
        const bool in_smem = (t1 - tb) <= OB_BYTES;          // else: this tile writes straight to global memory
        uint8_t* const wbase = in_smem ? S.ob - tb : P.out;  // byte x of the output is written at wbase + x
        const uint8_t* lit = P.comp + B.lit_off;
        // ---- phase 0: literal runs (a4); validate matches (I2) and remember them in registers
#pragma unroll
        for (int k = 0; k < PRE_ITEMS; ++k) {
            bool ok = (uint64_t)pos + c[k] + l[k] <= B.raw_len && (uint64_t)lsrc + c[k] <= B.n_lit;
            if (!ok && (c[k] | l[k])) raise_fault(P.status, F_BLOCK_SUM, b);
            const uint32_t cc = ok ? c[k] : 0;
            if (cc && cc <= 16) { uint8_t* q = wbase + blk_lo + pos; for (uint32_t i = 0; i < cc; ++i) q[i] = lit[lsrc + i]; }
            uint32_t longm = __ballot_sync(0xFFFFFFFFu, cc > 16);
            while (longm) {
                const int sl = __ffs(longm) - 1; longm &= longm - 1;
                const uint32_t p2 = __shfl_sync(0xFFFFFFFFu, pos, sl), s2 = __shfl_sync(0xFFFFFFFFu, lsrc, sl),
                               n2 = __shfl_sync(0xFFFFFFFFu, cc, sl);
                warp_copy(wbase + blk_lo + p2, lit + s2, n2, lane);
            }
            pos += c[k]; lsrc += c[k];
            bool m = ok && l[k] != 0;
            if (l[k] == 0 && (of[k] | dp[k])) raise_fault(P.status, F_PLACEHOLDER, b);
            const uint32_t mdst = blk_lo + pos;
            if (m) {
                if (of[k] >= mdst || l[k] < P.min_match) { raise_fault(P.status, F_SOURCE, b); m = false; }
                else if (dp[k] == 0 || dp[k] > P.max_depth) { raise_fault(P.status, F_DEPTH, b); m = false; }
            }
            if (m) { const uint32_t dist = mdst - of[k]; src_bytes += l[k] < dist ? l[k] : dist; }
            pos += l[k];
            c[k] = mdst;                                     // reuse c[] as the match destination
            if (!m) { l[k] = 0; dp[k] = 0; }
        }
        // ---- sort the tile's matches by depth into shared memory (a5, per tile): warp-ballot ranks
        {
            unsigned long long dm = 0ull;
#pragma unroll
            for (int k = 0; k < PRE_ITEMS; ++k) if (l[k]) dm |= 1ull << dp[k];
#pragma unroll
            for (int d = 16; d; d >>= 1) dm |= __shfl_xor_sync(0xFFFFFFFFu, dm, d);
            if (lane == 0 && dm) atomicOr(&S.depth_mask, dm);
            for (uint32_t d = 1; d <= P.max_depth; ++d) {
                uint32_t n = 0;
                if ((dm >> d) & 1ull) {
#pragma unroll
                    for (int k = 0; k < PRE_ITEMS; ++k) n += __popc(__ballot_sync(0xFFFFFFFFu, l[k] != 0 && dp[k] == d));
                }
                if (lane == 0) S.wcnt[warp][d] = (uint16_t)n;
            }
            __syncthreads();
            if (tid == 0) {                                  // depth-major exclusive scan over (depth, warp): <= 17 x 8 adds
                uint32_t run = 0;
                for (uint32_t d = 1; d <= P.max_depth; ++d) {
                    S.dstart[d] = run;
                    for (int w = 0; w < PRE_THREADS / 32; ++w) { const uint32_t n = S.wcnt[w][d]; S.wcnt[w][d] = (uint16_t)run; run += n; }
                    S.cnt[d] = run - S.dstart[d];
                }
                S.dstart[P.max_depth + 1] = run;
            }
            __syncthreads();
            for (uint32_t d = 1; d <= P.max_depth; ++d) {
                if (!((dm >> d) & 1ull)) continue;
                uint32_t at = S.wcnt[warp][d];
#pragma unroll
                for (int k = 0; k < PRE_ITEMS; ++k) {
                    const bool mine = l[k] != 0 && dp[k] == d;
                    const uint32_t m = __ballot_sync(0xFFFFFFFFu, mine);
                    if (mine) { const uint32_t i = at + __popc(m & ((1u << lane) - 1u)); S.e_dst[i] = c[k]; S.e_off[i] = of[k]; S.e_len[i] = (uint16_t)l[k]; }
                    at += __popc(m);
                }
            }
        }
        __syncthreads();
        if (in_smem) flush_tile(P.out, S.ob - tb, t0, t1);
        publish(P.prog, tile, 1u);
        const unsigned long long dmask = S.depth_mask;
        // per-depth match counts -> cursor[d] (k_check_cursors compares them with the header histogram)
        if (tid >= 1 && tid <= P.max_depth && S.cnt[tid]) atomicAdd(&P.cursor[tid], S.cnt[tid]);
        // ---- phases 1 .. max_depth: matches of depth d (a6), sequenced by the progress flags (a7)
        const uint8_t* const img = S.ob - tb;                // img + x = byte x of the output, if in_smem and x in [tb, t1)
        for (uint32_t d = 1; d <= P.max_depth; ++d) {
            if (!((dmask >> d) & 1ull)) continue;
            wait_ready(P, tile, d);
            const uint32_t e0 = S.dstart[d], e1 = S.dstart[d + 1];
            for (uint32_t base = e0 + warp * 64u; base < e1; base += (PRE_THREADS / 32) * 64u) {
                uint32_t md[2], so[2], ln[2];
                uint4 wa[2], wb[2];
                bool simple[2];
                const uint8_t* sp[2];
#pragma unroll
                for (int r = 0; r < 2; ++r) {
                    const uint32_t i = base + 32u * r + lane;
                    md[r] = 0; so[r] = 0; ln[r] = 0;
                    if (i < e1) { md[r] = S.e_dst[i]; so[r] = S.e_off[i]; ln[r] = S.e_len[i]; }
                    // a source that starts inside the tile is read from the shared image
                    sp[r] = (in_smem && so[r] >= t0) ? img + so[r] : (const uint8_t*)P.out + so[r];
                    simple[r] = ln[r] != 0 && ln[r] <= 16 && (md[r] - so[r]) >= ln[r];
                    const uint32_t sb = so[r] & 15u;
                    const uint4* p = reinterpret_cast<const uint4*>(sp[r] - sb);      // shared image keeps the output's alignment mod 16
                    wa[r] = make_uint4(0u, 0u, 0u, 0u); wb[r] = wa[r];
                    if (simple[r]) { wa[r] = p[0]; if (sb + ln[r] > 16) wb[r] = p[1]; }
                }
#pragma unroll
                for (int r = 0; r < 2; ++r) {
                    if (simple[r]) {
                        const uint32_t sb = so[r] & 15u, sh = (sb & 7u) * 8;
                        const unsigned long long a0 = (unsigned long long)wa[r].x | ((unsigned long long)wa[r].y << 32),
                                                 a1 = (unsigned long long)wa[r].z | ((unsigned long long)wa[r].w << 32),
                                                 b0 = (unsigned long long)wb[r].x | ((unsigned long long)wb[r].y << 32),
                                                 b1 = (unsigned long long)wb[r].z | ((unsigned long long)wb[r].w << 32);
                        const unsigned long long x0 = sb < 8 ? a0 : a1, x1 = sb < 8 ? a1 : b0, x2 = sb < 8 ? b0 : b1;
                        V16 v;
                        if (sh) { v.lo = (x0 >> sh) | (x1 << (64 - sh)); v.hi = (x1 >> sh) | (x2 << (64 - sh)); } else { v.lo = x0; v.hi = x1; }
                        store16(wbase + md[r], v, ln[r]);
                    } else if (ln[r] != 0 && ln[r] <= SHORT_MAX) thread_copy(wbase + md[r], sp[r], ln[r], md[r] - so[r]);
                }
#pragma unroll
                for (int r = 0; r < 2; ++r) {
                    uint32_t longm = __ballot_sync(0xFFFFFFFFu, ln[r] > SHORT_MAX);
                    while (longm) {
                        const int sl = __ffs(longm) - 1; longm &= longm - 1;
                        const uint32_t d2 = __shfl_sync(0xFFFFFFFFu, md[r], sl), o2 = __shfl_sync(0xFFFFFFFFu, so[r], sl),
                                       n2 = __shfl_sync(0xFFFFFFFFu, ln[r], sl);
                        const bool ssm = in_smem && o2 >= t0;
                        const uint8_t* sp2 = ssm ? img + o2 : (const uint8_t*)P.out + o2;
                        warp_match(wbase + d2, sp2, n2, d2 - o2, ssm || !in_smem, lane);
                    }
                }
            }
            __syncthreads();
            if (in_smem) flush_tile(P.out, S.ob - tb, t0, t1);
            publish(P.prog, tile, d + 1u);
        }
        publish(P.prog, tile, P.max_depth + 1u);
    }
#pragma unroll
    for (int d = 16; d; d >>= 1) src_bytes += __shfl_xor_sync(0xFFFFFFFFu, src_bytes, d);
    if (lane == 0 && src_bytes) atomicAdd(&P.status->match_src_bytes, src_bytes);
}

size_t fused_smem_bytes() { return sizeof(FusedSmem); }

cudaError_t fused_configure() {
    return cudaFuncSetAttribute(k_fused, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(FusedSmem));
}

int fused_max_ctas_per_sm() {
    int n = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k_fused, PRE_THREADS, sizeof(FusedSmem)) != cudaSuccess) return 0;
    return n;
}

void launch_fused(const Params& P, int grid, cudaStream_t st) {
    if (P.n_tiles) k_fused<<<grid, PRE_THREADS, sizeof(FusedSmem), st>>>(P);
}

}  // namespace ax
