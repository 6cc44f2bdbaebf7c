// k_pass.cu — strategy PASSES for shallow streams (e.g. the depth-limited encoder of PAPER.md:228 §7.4, "at most D
// match waves"): the token stream is parsed once per pass instead of being bucketed into wave lists:
//   k_pass 0    parse cmd[], len[] (a2) + scan inside the tile (a3) + literal scatter (a4).  Instance LISTING: also
//               reads dep[] / off[] and writes the wave lists of the SPARSE depths (Params::list_mask: depths holding
//               fewer than 1/8 of the sequences) — validation (I2), M_src, per-depth rank in shared memory, one global
//               atomic per depth and tile to reserve the tile's slice of the list (a5 for those depths only).
//   k_pass p    parse + scan + validation (I2), M_src and copy of the matches with dep == p (a6), one launch per DENSE
//               depth (a7: a kernel boundary orders wave p-1 before wave p); sparse depths are copied from
//               their lists by k_waves (k_match.cu), in depth order with the passes.  A match whose dep is 0 or above
//               max_depth is copied by nothing and shows up as a histogram mismatch (F_DEPTH).
//   k_litcopy   the queued long literal runs (a4), eight lanes per piece, over the whole grid.
// Why: with few waves, lists for everything cost more than they save — 10 B written + 10 B read per
// match and a bucketing kernel (k_pre) that ranks, reserves and scatters every match — whereas re-reading the
// 10 B/sequence stream is a pure streaming read with no inter-CTA dependency: tiles are assigned statically, their
// prefixes inside the block come from k_tilesum.  A sweep costs ~0.65 ms per 176 M sequences before it copies a byte,
// so it pays only for a depth that holds many matches; hence the lists for the sparse ones.
// Matches are copied exactly as in the wave kernel (copy.cuh: register funnel shift, OR-merge into the zeroed output).
#include "common.cuh"
#include "copy.cuh"

namespace ax {

constexpr int PS_WARPS = PS_THREADS / 32;
constexpr int PS_WCAP = 32 * PRE_ITEMS;                  // matches one warp can select in a tile (256)

struct PassSmem {
    unsigned long long warp_sum[PS_WARPS];
    uint32_t cnt;                                        // matches this CTA copied in this pass (histogram check)
    uint32_t lcnt[PASS_MAX_DEPTH + 1], lbase[PASS_MAX_DEPTH + 1];   // literal pass: the tile's listed matches per sparse depth, their list slots
    uint32_t lloc[PASS_MAX_DEPTH + 1], nloc;             // ... and their places in the tile's staging area (w_dst / w_off / w_len / e_g)
    uint32_t e_g[TILE_STREAM];                           // list slot of every staged entry
    uint32_t w_dst[PS_WARPS][PS_WCAP];                   // per warp: the tile's matches of this pass, compacted
    uint32_t w_off[PS_WARPS][PS_WCAP];
    uint16_t w_len[PS_WARPS][PS_WCAP];
};

// ---- pass p: 0 = literals (LISTING: and the wave lists of the sparse depths), p >= 1 = matches of depth p
template <bool LIT, bool LISTING, bool VECLIT>
__global__ void __launch_bounds__(PS_THREADS, 1024 / PS_THREADS) k_pass(Params P, uint32_t p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    PassSmem& S = *reinterpret_cast<PassSmem*>(smem_raw);
    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    unsigned long long src_bytes = 0;
    if (P.status->fault_flags & F_INDEX) return;                    // the block index is inconsistent (k_index): touch nothing
    if (!LIT && P.status->fault_flags != 0) return;                 // a faulty stream is flagged, not decoded further
    if (tid == 0) S.cnt = 0;
    constexpr bool listing = LIT && LISTING;                        // some depths are sparse: their matches are listed here
    if (listing && tid <= PASS_MAX_DEPTH) S.lcnt[tid] = 0;
    if (listing && tid == 0) S.nloc = 0;
    __syncthreads();
    for (uint32_t tile = blockIdx.x; tile < P.n_tiles; tile += gridDim.x) {
        const uint32_t b = P.tile_blk[tile];
        const unsigned long long pre = P.tile_state[tile];
        const BlockDesc B = P.blocks[b];
        const uint32_t j0 = (tile - B.tile_base) * TILE_STREAM + tid * PRE_ITEMS;
        // ---- a2: parse (pass 0 needs neither depths nor sources)
        Seq8 q;
        load_seq8(q, P.comp, B, j0, !LIT || listing);
        uint32_t (&c)[PRE_ITEMS] = q.c, (&l)[PRE_ITEMS] = q.l, (&dp)[PRE_ITEMS] = q.dp, (&of)[PRE_ITEMS] = q.of;
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
            // copies the match: pass 0 reads only cmd[], len[] and lit[]).  Runs of up to LONG_LIT bytes: one thread, byte by
            // byte (the typical run on compressible data is 1-2 bytes); longer runs: queued for k_litcopy, which spreads
            // them over the whole grid with 16-byte vector stores.
            const uint8_t* lit = P.comp + B.lit_off;
            uint8_t* outb = P.out + B.out_base;
            const uint32_t pos0 = pos;
            uint32_t rank[PRE_ITEMS], sel_mask = 0;                  // (listing) rank of a listed match among its depth's in the tile
#pragma unroll
            for (int k = 0; k < PRE_ITEMS; ++k) {
                const bool ok = (uint64_t)pos + c[k] + l[k] <= B.raw_len && (uint64_t)lsrc + c[k] <= B.n_lit;
                rank[k] = 0;
                if (listing && ok && l[k] != 0 && dp[k] <= PASS_MAX_DEPTH && ((P.list_mask >> dp[k]) & 1u)) {
                    const uint32_t mdst = blk_lo + pos + c[k];
                    if (of[k] >= mdst || l[k] < P.min_match) raise_fault(P.status, F_SOURCE, b);              // I2
                    else {
                        const uint32_t dist = mdst - of[k];
                        src_bytes += l[k] < dist ? l[k] : dist;
                        rank[k] = atomicAdd(&S.lcnt[dp[k]], 1u); sel_mask |= 1u << k;
                    }
                }
                if (!ok && (c[k] | l[k])) raise_fault(P.status, F_BLOCK_SUM, b);
                const uint32_t cc = ok ? c[k] : 0;
                if (__any_sync(0xFFFFFFFFu, cc != 0)) {  // literal runs are rare on compressible data: skip as a warp
                    if (VECLIT && cc > 4 && cc <= LONG_LIT) store16(outb + pos, load16(lit + lsrc, cc), cc);   // (streams of longer runs)
                    else if (cc && cc <= LONG_LIT) { for (uint32_t i = 0; i < cc; ++i) outb[pos + i] = lit[lsrc + i]; }   // typical run: 1-2 bytes
                    queue_long_literals(P, cc > LONG_LIT, blk_lo + pos, B.lit_off + lsrc, cc, lane, b);       // copied by k_litcopy
                }
                pos += c[k] + l[k]; lsrc += c[k];
            }
            if (listing) {
                // a5 for the sparse depths only: reserve the tile's slice of each depth's wave list, group the tile's entries by
                // depth in shared memory (the staging arrays of the match passes are idle here), then write them out in list
                // order so that consecutive threads store consecutive slots (as k_pre does: coalesced runs, one per depth)
                uint32_t* const e_dst = &S.w_dst[0][0]; uint32_t* const e_off = &S.w_off[0][0]; uint16_t* const e_len = &S.w_len[0][0];
                __syncthreads();
                if (tid <= PASS_MAX_DEPTH && S.lcnt[tid]) {
                    S.lbase[tid] = atomicAdd(&P.cursor[tid], S.lcnt[tid]);
                    S.lloc[tid] = atomicAdd(&S.nloc, S.lcnt[tid]);
                }
                __syncthreads();
                uint32_t p2 = pos0;
#pragma unroll
                for (int k = 0; k < PRE_ITEMS; ++k) {
                    p2 += c[k];
                    if (sel_mask & (1u << k)) {
                        const uint32_t i = S.lloc[dp[k]] + rank[k];
                        uint32_t g = S.lbase[dp[k]] + rank[k];
                        if (g >= P.wave_off[dp[k] + 1]) { raise_fault(P.status, F_DEPTH, b); g = 0xFFFFFFFFu; }   // more matches than the histogram says
                        e_dst[i] = blk_lo + p2; e_off[i] = of[k]; e_len[i] = (uint16_t)l[k]; S.e_g[i] = g;
                    }
                    p2 += l[k];
                }
                __syncthreads();
                const uint32_t nloc = S.nloc;
                for (uint32_t i = tid; i < nloc; i += PS_THREADS) {
                    const uint32_t g = S.e_g[i];
                    if (g != 0xFFFFFFFFu) { P.wl_dst[g] = e_dst[i]; P.wl_off[g] = e_off[i]; P.wl_len[g] = e_len[i]; }
                }
                __syncthreads();
                if (tid <= PASS_MAX_DEPTH) S.lcnt[tid] = 0;          // (ordered before the next tile's counting by its scan barriers)
                if (tid == 0) S.nloc = 0;
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
            if (lane == 0 && at) atomicAdd(&S.cnt, at);
            __syncwarp();
            // one entry per lane and step (measured on text1g_d4: 3.99 / 4.16 / 4.74 ms for 1 / 2 / 4 entries per lane)
            for (uint32_t base = 0; base < at; base += 32) {
                Ent e[1];
                const uint32_t i = base + lane;
                e[0].mdst = 0; e[0].off = 0; e[0].len = 0;
                if (i < at) { e[0].mdst = S.w_dst[warp][i]; e[0].off = S.w_off[warp][i]; e[0].len = S.w_len[warp][i]; }
                copy_ents<1>(P.out, e, lane);
            }
            __syncwarp();
        }
    }
    if (!LIT) {
        __syncthreads();
        if (tid == 0 && S.cnt) atomicAdd(&P.cursor[p], S.cnt);      // histogram check (k_check_cursors after the last pass)
    }
    if (!LIT || listing) {
#pragma unroll
        for (int d = 16; d; d >>= 1) src_bytes += __shfl_xor_sync(0xFFFFFFFFu, src_bytes, d);
        if (lane == 0 && src_bytes) atomicAdd(LIT ? &P.status->src_bytes_pre : &P.status->match_src_bytes, src_bytes);
    }
}

// Before the match passes of a step: the counters they accumulate start from the header's offsets again, so that
// PHASE_MATCH can be replayed on its own (this is how the match phase is timed alone).
__global__ void k_pass_reset(Params P) {
    const uint32_t d = blockIdx.x * blockDim.x + threadIdx.x;
    if (d == 0) P.status->match_src_bytes = 0ull;
    if (d >= 1 && d <= P.max_depth && !((P.list_mask >> d) & 1u)) P.cursor[d] = P.wave_off[d];   // (listed depths were counted by PRE)
}

void launch_pass_reset(const Params& P, cudaStream_t st) {
    k_pass_reset<<<(P.max_depth + 256) / 256, 256, 0, st>>>(P);
}

cudaError_t pass_configure() {
    const int n = (int)sizeof(PassSmem);
    cudaError_t e = cudaFuncSetAttribute(k_pass<false, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, n);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_pass<true, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, n);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_pass<true, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, n);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_pass<true, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, n);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_pass<true, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, n);
    return e;
}

int pass_max_ctas_per_sm() {
    int n = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k_pass<false, false, false>, PS_THREADS, sizeof(PassSmem)) != cudaSuccess) return 0;
    return n;
}

// ---- step a4, the queued pieces of long literal runs: eight lanes per piece (x 16 bytes per step), pieces strided over all
// lane groups of the grid, so that thousands of independent copies are in flight
constexpr int LC_THREADS = 256;
__global__ void __launch_bounds__(LC_THREADS) k_litcopy(Params P) {
    if (P.status->fault_flags & (F_INDEX | F_BLOCK_SUM)) return;
    uint32_t n = P.status->lit_q_count;
    if (n > P.lit_q_cap) n = P.lit_q_cap;
    constexpr uint32_t G = 8;                       // lanes per piece (x 16 bytes per step): 8 / 16 measured on runs of ~260 B
    const uint32_t hw = (blockIdx.x * LC_THREADS + threadIdx.x) / G, nhw = (gridDim.x * LC_THREADS) / G, l16 = threadIdx.x % G;
    for (uint32_t i = hw; i < n; i += nhw) {
        const uint4 e = P.lit_q[i];
        group_copy<G>(P.out + e.x, P.comp + (((unsigned long long)e.w << 32) | e.z), e.y, l16);
    }
}

void launch_litcopy(const Params& P, int grid, cudaStream_t st) {
    if (P.lit_q_cap) k_litcopy<<<grid, LC_THREADS, 0, st>>>(P);
}

void launch_pass(const Params& P, uint32_t p, int grid, cudaStream_t st) {
    if (!P.n_tiles) return;
    const uint32_t g = (uint32_t)grid < P.n_tiles ? grid : P.n_tiles;
    // Literal pass: the instance is picked from the header — with sparse depths it also lists them; where the mean literal run
    // is 4-20 bytes, runs of 5-16 bytes go through one 16-byte register value instead of the byte loop (separate instances,
    // so that the common one — runs of 1-2 bytes — keeps its short unrolled token loop: DESIGN.md 6.7).
    if (p == 0 && P.list_mask && P.long_runs) k_pass<true, true, true><<<g, PS_THREADS, sizeof(PassSmem), st>>>(P, p);
    else if (p == 0 && P.list_mask) k_pass<true, true, false><<<g, PS_THREADS, sizeof(PassSmem), st>>>(P, p);
    else if (p == 0 && P.long_runs) k_pass<true, false, true><<<g, PS_THREADS, sizeof(PassSmem), st>>>(P, p);
    else if (p == 0) k_pass<true, false, false><<<g, PS_THREADS, sizeof(PassSmem), st>>>(P, p);
    else k_pass<false, false, false><<<g, PS_THREADS, sizeof(PassSmem), st>>>(P, p);
}

}  // namespace ax
