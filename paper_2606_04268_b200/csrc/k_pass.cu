// k_pass.cu — strategy PASSES for shallow streams (AUTO: max_depth <= 8; accepted up to 16; e.g. the depth-limited encoder of
// PAPER.md:228 §7.4): no wave lists at all.  The token stream is parsed once per pass instead:
//   k_tilesum   one CTA per 1 MB block walks the block's tiles (2048 sequences each) and writes, per tile, the
//               exclusive prefix of (cmd+len, cmd) inside the block (a3, the block-level part of the scan) and the
//               tile's block index; checks that the block sums to raw_len / n_lit (invariant I1).
//   k_pass 0    parse cmd[], len[] (a2) + scan inside the tile (a3) + literal scatter (a4).
//   k_pass p    parse + scan + validation (I2), M_src and copy of the matches with dep == p (a6), p = 1 .. max_depth,
//               one launch each (a7: a kernel boundary orders wave p-1 before wave p); a match whose
//               dep is 0 or above max_depth is copied by no pass and shows up as a histogram mismatch (F_DEPTH).
// Why: with few waves the wave lists cost more than they save — 10 B written + 10 B read per match
// and a bucketing kernel (k_pre) that ranks, reserves and scatters every match at ~1 TB/s —
// whereas re-reading the 10 B/sequence stream is a pure streaming read with no inter-CTA dependency: tiles are
// assigned statically, prefixes come from k_tilesum, nothing is reserved with atomics.
// Matches are copied exactly as in the wave kernel (copy.cuh: register funnel shift, OR-merge into the zeroed output).
#include "common.cuh"
#include "copy.cuh"

namespace ax {

constexpr int PS_WARPS = PRE_THREADS / 32;
constexpr int PS_WCAP = 32 * PRE_ITEMS;                  // matches one warp can select in a tile (256)

struct PassSmem {
    unsigned long long warp_sum[PS_WARPS];
    uint32_t cnt[FUSED_MAX_DEPTH + 2];
    uint32_t w_dst[PS_WARPS][PS_WCAP];                   // per warp: the tile's matches of this pass, compacted
    uint32_t w_off[PS_WARPS][PS_WCAP];
    uint16_t w_len[PS_WARPS][PS_WCAP];
};

// ---- per-tile exclusive prefixes inside each block; tile -> block map
// One CTA per block; each WARP sums whole tiles on its own (all its loads independent), then one warp scans the
// tile totals.  Blocks with more than TS_CHUNK tiles are walked in chunks with a carry.
constexpr uint32_t TS_CHUNK = 1024;

__global__ void __launch_bounds__(PRE_THREADS) k_tilesum(Params P) {
    __shared__ unsigned long long s_tot[TS_CHUNK];
    __shared__ unsigned long long s_carry;
    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    for (uint32_t b = blockIdx.x; b < P.n_blocks; b += gridDim.x) {
        const BlockDesc B = P.blocks[b];
        const uint32_t nt = (B.n_seq + TILE - 1) / TILE;
        __syncthreads();
        if (tid == 0) s_carry = 0;
        for (uint32_t t0 = 0; t0 < nt; t0 += TS_CHUNK) {
            const uint32_t tn = nt - t0 < TS_CHUNK ? nt - t0 : TS_CHUNK;
            for (uint32_t t = warp; t < tn; t += PS_WARPS) {
                unsigned long long s = 0;
#pragma unroll
                for (int r = 0; r < TILE / 256; ++r) {
                    const uint32_t j0 = (t0 + t) * TILE + r * 256 + lane * 8;
                    if (j0 < B.n_seq) {
                        const uint4 vc = *reinterpret_cast<const uint4*>(P.comp + B.cmd_off + 2ull * j0);
                        const uint4 vl = *reinterpret_cast<const uint4*>(P.comp + B.len_off + 2ull * j0);
                        const uint32_t wc[4] = {vc.x, vc.y, vc.z, vc.w}, wl[4] = {vl.x, vl.y, vl.z, vl.w};
#pragma unroll
                        for (int k = 0; k < 8; ++k) {
                            if (j0 + k < B.n_seq) {
                                const uint32_t c = (wc[k >> 1] >> (16 * (k & 1))) & 0xFFFFu, l = (wl[k >> 1] >> (16 * (k & 1))) & 0xFFFFu;
                                s += ((unsigned long long)(c + l) << 32) | c;
                            }
                        }
                    }
                }
#pragma unroll
                for (int d = 16; d; d >>= 1) s += __shfl_xor_sync(0xFFFFFFFFu, s, d);
                if (lane == 0) s_tot[t] = s;
            }
            __syncthreads();
            if (warp == 0) {                             // exclusive scan of the chunk's tile totals, 32 at a time
                unsigned long long run = s_carry;
                for (uint32_t i0 = 0; i0 < tn; i0 += 32) {
                    const uint32_t i = i0 + lane;
                    const unsigned long long v = i < tn ? s_tot[i] : 0ull;
                    unsigned long long inc = v;
#pragma unroll
                    for (int d = 1; d < 32; d <<= 1) {
                        const unsigned long long x = __shfl_up_sync(0xFFFFFFFFu, inc, d);
                        if (lane >= d) inc += x;
                    }
                    unsigned long long ex = run + inc - v;
                    if ((ex >> 32) > 0x7FFFFFFFull) ex = (0x7FFFFFFFull << 32) | (uint32_t)ex;   // saturate (corrupt stream)
                    if (i < tn) { P.tile_state[B.tile_base + t0 + i] = ex; P.prog[B.tile_base + t0 + i] = b; }
                    run += __shfl_sync(0xFFFFFFFFu, inc, 31);
                    if ((run >> 32) > 0x7FFFFFFFull) run = (0x7FFFFFFFull << 32) | (uint32_t)run;
                }
                if (lane == 0) s_carry = run;
            }
            __syncthreads();
        }
        if (tid == 0 && ((uint32_t)(s_carry >> 32) != B.raw_len || (uint32_t)s_carry != B.n_lit)) raise_fault(P.status, F_BLOCK_SUM, b);
    }
}

// ---- pass p: 0 = literals + validation, p >= 1 = matches of depth p
template <bool LIT>   // LIT: pass 0 (literals); otherwise p >= 1
__global__ void __launch_bounds__(PRE_THREADS, 4) k_pass(Params P, uint32_t p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    PassSmem& S = *reinterpret_cast<PassSmem*>(smem_raw);
    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    unsigned long long src_bytes = 0;
    if (!LIT && P.status->fault_flags != 0) return;                 // a faulty stream is flagged, not decoded further
    if (tid <= FUSED_MAX_DEPTH) S.cnt[tid] = 0;
    __syncthreads();
    for (uint32_t tile = blockIdx.x; tile < P.n_tiles; tile += gridDim.x) {
        const uint32_t b = P.prog[tile];
        const unsigned long long pre = P.tile_state[tile];
        const BlockDesc B = P.blocks[b];
        const uint32_t j0 = (tile - B.tile_base) * TILE + tid * PRE_ITEMS;
        // ---- a2: parse
        uint32_t c[PRE_ITEMS], l[PRE_ITEMS], dp[PRE_ITEMS], of[PRE_ITEMS];
        if (j0 < B.n_seq) {
            const uint4 vc = *reinterpret_cast<const uint4*>(P.comp + B.cmd_off + 2ull * j0);
            const uint4 vl = *reinterpret_cast<const uint4*>(P.comp + B.len_off + 2ull * j0);
            uint4 vd = make_uint4(0u, 0u, 0u, 0u), o0 = vd, o1 = vd;
            if (!LIT) {                                  // pass 0 (literals) needs neither depths nor sources
                vd = *reinterpret_cast<const uint4*>(P.comp + B.dep_off + 2ull * j0);
                o0 = *reinterpret_cast<const uint4*>(P.comp + B.off_off + 4ull * j0);
                o1 = *reinterpret_cast<const uint4*>(P.comp + B.off_off + 4ull * j0 + 16);
            }
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
        // ---- a3: scan inside the tile; the block-level prefix comes from k_tilesum.  The literal pass scans the pair
        // (cmd+len, cmd) packed in one u64; match passes need output positions only (32-bit shuffles)
        uint32_t pos, lsrc = 0;
        if (LIT) {
            unsigned long long tsum = 0;
#pragma unroll
            for (int k = 0; k < PRE_ITEMS; ++k) tsum += ((unsigned long long)(c[k] + l[k]) << 32) | c[k];
            unsigned long long inc = tsum;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const unsigned long long t = __shfl_up_sync(0xFFFFFFFFu, inc, d);
                if (lane >= d) inc += t;
            }
            __syncthreads();                             // previous tile's readers of warp_sum are done
            if (lane == 31) S.warp_sum[warp] = inc;
            __syncthreads();
            unsigned long long wpre = 0;
#pragma unroll
            for (int w = 0; w < PS_WARPS; ++w) if (w < (int)warp) wpre += S.warp_sum[w];
            const unsigned long long ex = pre + wpre + (inc - tsum);
            pos = (uint32_t)(ex >> 32);                  // output offset inside the block
            lsrc = (uint32_t)ex;                         // offset inside the block's lit[]
        } else {
            uint32_t tsum = 0;
#pragma unroll
            for (int k = 0; k < PRE_ITEMS; ++k) tsum += c[k] + l[k];
            uint32_t inc = tsum;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const uint32_t t = __shfl_up_sync(0xFFFFFFFFu, inc, d);
                if (lane >= d) inc += t;
            }
            __syncthreads();
            if (lane == 31) S.warp_sum[warp] = inc;
            __syncthreads();
            uint32_t wpre = 0;
#pragma unroll
            for (int w = 0; w < PS_WARPS; ++w) if (w < (int)warp) wpre += (uint32_t)S.warp_sum[w];
            pos = (uint32_t)(pre >> 32) + wpre + (inc - tsum);
        }
        const uint32_t blk_lo = (uint32_t)B.out_base;
        if (LIT) {
            // ---- a4 literal scatter (token validation, M_src and the per-depth counts are taken by the pass that
            // copies the match: pass 0 reads only cmd[], len[] and lit[])
            const uint8_t* lit = P.comp + B.lit_off;
            uint8_t* outb = P.out + B.out_base;
#pragma unroll
            for (int k = 0; k < PRE_ITEMS; ++k) {
                const bool ok = (uint64_t)pos + c[k] + l[k] <= B.raw_len && (uint64_t)lsrc + c[k] <= B.n_lit;
                if (!ok && (c[k] | l[k])) raise_fault(P.status, F_BLOCK_SUM, b);
                const uint32_t cc = ok ? c[k] : 0;
                if (cc && cc <= 16) { for (uint32_t i = 0; i < cc; ++i) outb[pos + i] = lit[lsrc + i]; }
                uint32_t longm = __ballot_sync(0xFFFFFFFFu, cc > 16);
                while (longm) {
                    const int sl = __ffs(longm) - 1; longm &= longm - 1;
                    const uint32_t p2 = __shfl_sync(0xFFFFFFFFu, pos, sl), s2 = __shfl_sync(0xFFFFFFFFu, lsrc, sl),
                                   n2 = __shfl_sync(0xFFFFFFFFu, cc, sl);
                    warp_copy(outb + p2, lit + s2, n2, lane);
                }
                pos += c[k] + l[k]; lsrc += c[k];
            }
        } else {
            // ---- a6: select this pass's matches (same validity rule as pass 0), compact them per warp, copy
            uint32_t at = 0, sb = 0;
#pragma unroll
            for (int k = 0; k < PRE_ITEMS; ++k) {
                const bool ok = (uint64_t)pos + c[k] + l[k] <= B.raw_len;
                pos += c[k];
                const uint32_t mdst = blk_lo + pos;
                bool sel = ok && l[k] != 0 && dp[k] == p;
                if (sel && (of[k] >= mdst || l[k] < P.min_match)) { raise_fault(P.status, F_SOURCE, b); sel = false; }   // I2
                if (p == 1 && l[k] == 0 && (of[k] | dp[k])) raise_fault(P.status, F_PLACEHOLDER, b);
                if (sel) { const uint32_t dist = mdst - of[k]; sb += l[k] < dist ? l[k] : dist; }
                const uint32_t msk = __ballot_sync(0xFFFFFFFFu, sel);
                if (sel) {
                    const uint32_t i = at + __popc(msk & ((1u << lane) - 1u));
                    S.w_dst[warp][i] = mdst; S.w_off[warp][i] = of[k]; S.w_len[warp][i] = (uint16_t)l[k];
                }
                at += __popc(msk);
                pos += l[k];
            }
            src_bytes += sb;
            if (lane == 0 && at) atomicAdd(&S.cnt[p], at);          // histogram check (k_check_cursors after the last pass)
            __syncwarp();
#ifndef AX_PASS_U
#define AX_PASS_U 1   /* measured on text1g_d4: match passes 3.99 / 4.16 / 4.74 ms for 1 / 2 / 4 entries per lane and step */
#endif
            for (uint32_t base = 0; base < at; base += 32 * AX_PASS_U) {
                Ent e[AX_PASS_U];
#pragma unroll
                for (int r = 0; r < AX_PASS_U; ++r) {
                    const uint32_t i = base + 32u * r + lane;
                    e[r].mdst = 0; e[r].off = 0; e[r].len = 0;
                    if (i < at) { e[r].mdst = S.w_dst[warp][i]; e[r].off = S.w_off[warp][i]; e[r].len = S.w_len[warp][i]; }
                }
                copy_ents<AX_PASS_U>(P.out, e, lane);
            }
            __syncwarp();
        }
    }
    if (!LIT) {
        __syncthreads();
        if (tid == 0 && S.cnt[p]) atomicAdd(&P.cursor[p], S.cnt[p]);
#pragma unroll
        for (int d = 16; d; d >>= 1) src_bytes += __shfl_xor_sync(0xFFFFFFFFu, src_bytes, d);
        if (lane == 0 && src_bytes) atomicAdd(&P.status->match_src_bytes, src_bytes);
    }
}

// Before the match passes of a step: the counters they accumulate start from the header's offsets again, so that
// PHASE_MATCH can be replayed on its own (this is how the match phase is timed alone).
__global__ void k_pass_reset(Params P) {
    const uint32_t d = blockIdx.x * blockDim.x + threadIdx.x;
    if (d == 0) P.status->match_src_bytes = 0ull;
    if (d >= 1 && d <= P.max_depth) P.cursor[d] = P.wave_off[d];
}

void launch_pass_reset(const Params& P, cudaStream_t st) {
    k_pass_reset<<<(P.max_depth + 256) / 256, 256, 0, st>>>(P);
}

cudaError_t pass_configure() {
    return cudaFuncSetAttribute(k_pass<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(PassSmem));
}

int pass_max_ctas_per_sm() {
    int n = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k_pass<false>, PRE_THREADS, sizeof(PassSmem)) != cudaSuccess) return 0;
    return n;
}

void launch_tilesum(const Params& P, int grid, cudaStream_t st) {
    if (P.n_blocks) k_tilesum<<<(uint32_t)grid < P.n_blocks ? grid : P.n_blocks, PRE_THREADS, 0, st>>>(P);
}

void launch_pass(const Params& P, uint32_t p, int grid, cudaStream_t st) {
    if (!P.n_tiles) return;
    const uint32_t g = (uint32_t)grid < P.n_tiles ? grid : P.n_tiles;
    if (p == 0) k_pass<true><<<g, PRE_THREADS, sizeof(PassSmem), st>>>(P, p);
    else k_pass<false><<<g, PRE_THREADS, sizeof(PassSmem), st>>>(P, p);
}

}  // namespace ax
