// k_pre.cu — steps a2-a5 fused: token parse, segmented exclusive length scan, literal scatter, depth bucketing.
//   a2  per sequence: lit_len = cmd[j], mlen = len[j]                                   (§3.2)
//   a3  dst[j] = out_base[b] + sum_{i<j}(cmd[i]+len[i]);  lsrc[j] = sum_{i<j} cmd[i]      (the sequential walk of
//       PAPER.md:53 restated as a scan; one independent scan per 1 MB block)
//   a4  out[dst[j] .. +cmd[j]) = lit_b[lsrc[j] ..)
//   a5  matches grouped by dep[j] into per-depth wave lists (mdst, off, len)             (§7.1)
// One tile = 2048 consecutive sequences of one block.  The block-level part of the scan (the prefix of each tile
// inside its block) is computed first by k_tilesum, so tiles are independent here: static assignment,
// no ticket, no look-back.  dst[] and lsrc[] are never written to memory.  Matches of depths 1 .. list_hi get list
// entries (list_hi = max_depth whenever this kernel runs).
#include "common.cuh"
#include "copy.cuh"

namespace ax {

struct PreSmem {
    unsigned long long warp_sum[PRE_THREADS / 32];
    uint32_t nloc;                       // entries placed in the tile's sorted list so far
    uint32_t e_dst[TILE_LIST], e_off[TILE_LIST], e_g[TILE_LIST];   // the tile's matches grouped by depth; e_g = index in the wave list
    uint16_t e_len[TILE_LIST];
    // followed in dynamic shared memory by the depth bins, sized to the stream (pre_bins(max_depth) entries each):
    //   uint32_t cnt[]    per-depth count inside the tile
    //   uint32_t gbase[]  per-depth start in the wave list reserved for this tile
    //   uint16_t lbase[]  per-depth start in the tile's sorted list (bins in reservation order)
};

__host__ __device__ inline uint32_t pre_bins(uint32_t max_depth) {       // 0 = deeper than the shared-memory bins
    return max_depth + 1 <= SMEM_DEPTHS ? ((max_depth + 1 + 7u) & ~7u) : 0u;
}
__host__ __device__ inline size_t pre_smem_for(uint32_t max_depth) {
    return ((sizeof(PreSmem) + 15) & ~(size_t)15) + (size_t)pre_bins(max_depth) * 10u;
}

__global__ void __launch_bounds__(PRE_THREADS, 1024 / PRE_THREADS) k_pre(Params P) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    PreSmem& S = *reinterpret_cast<PreSmem*>(smem_raw);
    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t nbins = pre_bins(P.max_depth);
    const bool smem_bins = nbins != 0;
    uint32_t* const s_cnt = reinterpret_cast<uint32_t*>(smem_raw + ((sizeof(PreSmem) + 15) & ~(size_t)15));
    uint32_t* const s_gbase = s_cnt + nbins;
    uint16_t* const s_lbase = reinterpret_cast<uint16_t*>(s_gbase + nbins);
    if (P.status->fault_flags & F_INDEX) return;          // the block index is inconsistent (k_index): touch nothing
    if (smem_bins) for (uint32_t i = tid; i <= P.max_depth; i += PRE_THREADS) s_cnt[i] = 0;
    unsigned long long src_bytes = 0;

    // Tiles are assigned statically; the per-tile prefix inside the block and the tile -> block map come from
    // k_tilesum, so there is no ticket, no look-back and no dependency between CTAs here.
    for (uint32_t tile = blockIdx.x; tile < P.n_tiles; tile += gridDim.x) {
        __syncthreads();
        if (tid == 0) S.nloc = 0;
        const uint32_t b = P.tile_blk[tile];
        const unsigned long long tile_prefix = P.tile_state[tile];
        const BlockDesc B = P.blocks[b];
        const uint32_t t_in_blk = tile - B.tile_base;
        const uint32_t j0 = t_in_blk * TILE_LIST + tid * PRE_ITEMS;          // first sequence of this thread
        // ---- a2: parse (16-byte loads; streams are padded to 16 bytes, entries past n_seq are masked)
        Seq8 q;
        load_seq8(q, P.comp, B, j0, true);
        uint32_t (&c)[PRE_ITEMS] = q.c, (&l)[PRE_ITEMS] = q.l, (&dp)[PRE_ITEMS] = q.dp, (&of)[PRE_ITEMS] = q.of;
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
        unsigned long long wpre = 0;
#pragma unroll
        for (int w = 0; w < PRE_THREADS / 32; ++w) {
            const unsigned long long x = S.warp_sum[w];
            if (w < (int)warp) wpre += x;
        }
        const unsigned long long ex = tile_prefix + wpre + (inc - tsum);
        uint32_t pos = (uint32_t)(ex >> 32);                 // output offset inside the block
        uint32_t lsrc = (uint32_t)ex;                        // offset inside the block's lit[]
        const uint8_t* lit = P.comp + B.lit_off;
        uint8_t* outb = P.out + B.out_base;
        // ---- a4 literal scatter + token validation (I2); c[] becomes the match destination, of[] = 0xFFFFFFFF marks
        // "no entry" (a valid off is < mdst <= 2^32-1)
        uint32_t rank[PRE_ITEMS];
        uint32_t first_mask = 0;                             // bit k: this thread opened depth bin dp[k] in this tile
#pragma unroll
        for (int k = 0; k < PRE_ITEMS; ++k) {
            const bool ok = (uint64_t)pos + c[k] + l[k] <= B.raw_len && (uint64_t)lsrc + c[k] <= B.n_lit;
            if (!ok && (c[k] | l[k])) raise_fault(P.status, F_BLOCK_SUM, b);
            const uint32_t cc = ok ? c[k] : 0;
            if (__any_sync(0xFFFFFFFFu, cc != 0)) {          // literal runs are rare on compressible data: skip as a warp
                if (cc && cc <= LONG_LIT) { for (uint32_t i = 0; i < cc; ++i) outb[pos + i] = lit[lsrc + i]; }   // typical run: 1-2 bytes
                queue_long_literals(P, cc > LONG_LIT, (uint32_t)B.out_base + pos, B.lit_off + lsrc, cc, lane, b);   // copied by k_litcopy
            }
            pos += c[k]; lsrc += c[k];
            bool m = ok && l[k] != 0;
            if (l[k] == 0 && (of[k] | dp[k])) raise_fault(P.status, F_PLACEHOLDER, b);
            const uint32_t mdst = (uint32_t)B.out_base + pos;
            if (m) {
                if (of[k] >= mdst || l[k] < P.min_match) { raise_fault(P.status, F_SOURCE, b); m = false; }
                else if (dp[k] == 0 || dp[k] > P.max_depth) { raise_fault(P.status, F_DEPTH, b); m = false; }
            }
            if (m) { const uint32_t dist = mdst - of[k]; src_bytes += l[k] < dist ? l[k] : dist; }
            of[k] = m ? of[k] : 0xFFFFFFFFu;
            c[k] = mdst;
            pos += l[k];
        }
        // ---- a5 ranking: one shared-memory atomic per match, all eight of a thread in flight at once (this kernel
        // serves streams of more than 8 depths, where a warp's 32 keys are mostly distinct)
#pragma unroll
        for (int k = 0; k < PRE_ITEMS; ++k) {
            rank[k] = 0;
            if (smem_bins) {
                if (of[k] != 0xFFFFFFFFu) rank[k] = atomicAdd(&s_cnt[dp[k]], 1u);
            } else {
                // streams deeper than the shared-memory bins: one GLOBAL atomic per distinct depth in the warp
                const bool m = of[k] != 0xFFFFFFFFu;
                const uint32_t peers = __match_any_sync(0xFFFFFFFFu, m ? dp[k] : 0u);
                const int leader = __ffs(peers) - 1;
                uint32_t base = 0;
                if (m && (int)lane == leader) base = atomicAdd(&P.cursor[dp[k]], (uint32_t)__popc(peers));
                base = __shfl_sync(0xFFFFFFFFu, base, leader);
                if (m) rank[k] = base + __popc(peers & ((1u << lane) - 1u));
            }
        }
        if (smem_bins) {
#pragma unroll
            for (int k = 0; k < PRE_ITEMS; ++k) if (of[k] != 0xFFFFFFFFu && rank[k] == 0) first_mask |= 1u << k;
        }
        if (smem_bins) {
            __syncthreads();
#pragma unroll
            for (int k = 0; k < PRE_ITEMS; ++k)
                if (first_mask & (1u << k)) {            // reserve this tile's slice of the depth's wave list
                    const uint32_t n = s_cnt[dp[k]];
                    const uint32_t g = atomicAdd(&P.cursor[dp[k]], n);
                    s_gbase[dp[k]] = g;
                    s_lbase[dp[k]] = (uint16_t)atomicAdd(&S.nloc, n);
                    s_cnt[dp[k]] = 0;                    // bin is clean again for the next tile
                }
            __syncthreads();
            // ---- a5: group the tile's entries by depth in shared memory, then write them out in list order so
            // that consecutive threads store consecutive list slots (coalesced runs, one per depth present)
#pragma unroll
            for (int k = 0; k < PRE_ITEMS; ++k) {
                if (of[k] == 0xFFFFFFFFu) continue;
                const uint32_t i = (uint32_t)s_lbase[dp[k]] + rank[k];
                uint32_t g = s_gbase[dp[k]] + rank[k];
                if (g >= P.wave_off[dp[k] + 1]) { raise_fault(P.status, F_DEPTH, b); g = 0xFFFFFFFFu; }   // more matches than the histogram says
                S.e_dst[i] = c[k]; S.e_off[i] = of[k]; S.e_len[i] = (uint16_t)l[k]; S.e_g[i] = g;
            }
            __syncthreads();
            const uint32_t nloc = S.nloc;
            for (uint32_t i = tid; i < nloc; i += PRE_THREADS) {
                const uint32_t g = S.e_g[i];
                if (g != 0xFFFFFFFFu) { P.wl_dst[g] = S.e_dst[i]; P.wl_off[g] = S.e_off[i]; P.wl_len[g] = S.e_len[i]; }
            }
        } else {
            // ---- a5 (streams deeper than the shared-memory bins): ranks came from global cursors, write directly
#pragma unroll
            for (int k = 0; k < PRE_ITEMS; ++k) {
                if (of[k] == 0xFFFFFFFFu) continue;
                const uint32_t at = rank[k];
                if (at >= P.wave_off[dp[k] + 1]) { raise_fault(P.status, F_DEPTH, b); continue; }
                P.wl_dst[at] = c[k]; P.wl_off[at] = of[k]; P.wl_len[at] = (uint16_t)l[k];
            }
        }
    }
    // ---- M_src for the roofline report (aceapex_stats.match_src_bytes)
#pragma unroll
    for (int d = 16; d; d >>= 1) src_bytes += __shfl_xor_sync(0xFFFFFFFFu, src_bytes, d);
    if (lane == 0 && src_bytes) atomicAdd(&P.status->match_src_bytes, src_bytes);
}

// After PRE: every cursor must have reached the end of its list, else the histogram lied (fault F_DEPTH).
__global__ void k_check_cursors(Params P) {
    const uint32_t d = blockIdx.x * blockDim.x + threadIdx.x + 1;
    if (d <= P.list_hi && P.cursor[d] != P.wave_off[d + 1]) raise_fault(P.status, F_DEPTH, 0xFFFFFFFEu);
}


size_t pre_smem_bytes(uint32_t max_depth) { return pre_smem_for(max_depth); }

cudaError_t pre_configure() {
    return cudaFuncSetAttribute(k_pre, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pre_smem_for(SMEM_DEPTHS - 1));
}

int pre_max_ctas_per_sm(uint32_t max_depth) {
    int n = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k_pre, PRE_THREADS, pre_smem_for(max_depth)) != cudaSuccess) return 0;
    return n;
}

void launch_check_cursors(const Params& P, cudaStream_t st) {
    if (P.list_hi) k_check_cursors<<<(P.list_hi + 255) / 256, 256, 0, st>>>(P);
}

void launch_pre(const Params& P, int grid, cudaStream_t st) {
    if (P.n_tiles) k_pre<<<grid, PRE_THREADS, pre_smem_for(P.max_depth), st>>>(P);
    launch_check_cursors(P, st);
}

}  // namespace ax
