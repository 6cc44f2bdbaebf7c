// k_index.cu — step a1 (block index) of the ACEAPEX GPU decode ("Each 1 MB block is encoded as
// four separate arrays"; docs/FORMAT.md directory).  Reads header + directory + depth histogram from the
// device-resident compressed buffer and writes, into scratch: one BlockDesc per block (stream addresses,
// n_seq, n_lit, raw_len, first tile), the per-depth wave list offsets (exclusive prefix of the histogram's
// match counts) and the bucket cursors; clears the status words.
// The plan validated the same directory on the HOST copy; the device copy is a different buffer and may differ,
// so everything that later sizes an access is re-checked here against what the plan derived (comp_bytes, n_tiles,
// n_list): any disagreement raises F_INDEX and every later kernel of the decode returns at once.
#include "common.cuh"

namespace ax {

constexpr int IDX_THREADS = 1024;

// Exclusive block-wide scan of one value per thread (1024 threads); returns the exclusive prefix, total in *tot.
__device__ __forceinline__ uint32_t block_excl_scan(uint32_t v, uint32_t* s_warp, uint32_t* tot) {
    const uint32_t lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    uint32_t inc = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        uint32_t t = __shfl_up_sync(0xFFFFFFFFu, inc, d);
        if (lane >= d) inc += t;
    }
    if (lane == 31) s_warp[w] = inc;
    __syncthreads();
    if (w == 0) {
        uint32_t x = s_warp[lane], xi = x;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            uint32_t t = __shfl_up_sync(0xFFFFFFFFu, xi, d);
            if (lane >= d) xi += t;
        }
        s_warp[lane] = xi - x;
        if (lane == 31) s_warp[32] = xi;
    }
    __syncthreads();
    const uint32_t ex = s_warp[w] + inc - v;
    *tot = s_warp[32];
    __syncthreads();
    return ex;
}

__global__ void __launch_bounds__(IDX_THREADS) k_index(Params P) {
    __shared__ uint32_t s_warp[33];
    const uint8_t* dir = P.comp + HDR_BYTES;
    const uint8_t* hist = dir + (uint64_t)DIR_BYTES * P.n_blocks;
    if (threadIdx.x == 0) {
        P.status->fault_flags = 0; P.status->fault_block = 0xFFFFFFFFu; P.status->match_src_bytes = 0ull; P.status->src_bytes_pre = 0ull;
        P.status->n_final = 0; P.status->lit_q_count = 0; P.status->barrier = 0;
    }
    __syncthreads();
    const uint64_t meta = (HDR_BYTES + (uint64_t)DIR_BYTES * P.n_blocks + (uint64_t)HIST_BYTES * (P.max_depth + 1ull) + 127ull) & ~127ull;
    // ---- block descriptors + tile_base = exclusive prefix of ceil(n_seq / tile)
    uint32_t carry = 0;
    for (uint32_t b0 = 0; b0 < P.n_blocks; b0 += IDX_THREADS) {
        const uint32_t b = b0 + threadIdx.x;
        uint32_t ns = 0, nl = 0, nt = 0; uint64_t po = 0;
        bool ok = true;
        if (b < P.n_blocks) {
            const uint4 e = *reinterpret_cast<const uint4*>(dir + (uint64_t)DIR_BYTES * b);
            po = (uint64_t)e.x | ((uint64_t)e.y << 32); ns = e.z; nl = e.w;
            const uint64_t bytes = 3 * pad16(2ull * ns) + pad16(4ull * ns) + pad16(nl);
            ok = !(po & 127) && po >= meta && ns != 0 && po <= P.comp_bytes && bytes <= P.comp_bytes - po;
            if (!ok) { raise_fault(P.status, F_INDEX, b); ns = 0; }
            nt = (ns + P.tile - 1) / P.tile;
        }
        uint32_t tot;
        const uint32_t ex = block_excl_scan(nt, s_warp, &tot);
        if (b < P.n_blocks) {
            BlockDesc d;
            d.cmd_off = po;
            d.len_off = d.cmd_off + pad16(2ull * ns);
            d.dep_off = d.len_off + pad16(2ull * ns);
            d.off_off = d.dep_off + pad16(2ull * ns);
            d.lit_off = d.off_off + pad16(4ull * ns);
            d.out_base = (uint64_t)b * P.block_size;
            const uint64_t rem = P.raw_size - d.out_base;
            d.raw_len = rem < P.block_size ? (uint32_t)rem : P.block_size;
            d.n_seq = ns; d.n_lit = nl; d.tile_base = carry + ex;
            if (ok && (uint64_t)d.tile_base + nt > P.n_tiles) { raise_fault(P.status, F_INDEX, b); d.n_seq = 0; }
            P.blocks[b] = d;
        }
        carry += tot;
    }
    if (threadIdx.x == 0 && carry != P.n_tiles) raise_fault(P.status, F_INDEX, 0xFFFFFFFEu);
    // ---- wave list offsets: wave_off[d] = number of matches at depths 1 .. d-1 (d = 1 .. max_depth + 1)
    carry = 0;
    const uint32_t nd = P.max_depth + 2;                   // entries 0 .. max_depth + 1
    for (uint32_t d0 = 0; d0 < nd; d0 += IDX_THREADS) {
        const uint32_t d = d0 + threadIdx.x;
        uint32_t c = 0;                                    // count of depth d-1 feeds entry d; depth 0 holds literal runs
        if (d >= 2 && d < nd) c = *reinterpret_cast<const uint32_t*>(hist + (uint64_t)HIST_BYTES * (d - 1));
        uint32_t tot;
        const uint32_t ex = block_excl_scan(c, s_warp, &tot);
        if (d < nd) {
            uint32_t v = carry + ex + c;
            if (v < carry || (d == P.list_hi + 1 && v != P.n_list)) { raise_fault(P.status, F_INDEX, 0xFFFFFFFEu); }
            if (d <= P.list_hi + 1 && v > P.n_list) v = P.n_list;   // (faulted above or below: keeps every list index inside the lists)
            P.wave_off[d] = v; P.cursor[d] = v;
        }
        if (carry + tot < carry) raise_fault(P.status, F_INDEX, 0xFFFFFFFEu);
        carry += tot;
    }
}

void launch_index(const Params& P, cudaStream_t st) { k_index<<<1, IDX_THREADS, 0, st>>>(P); }

}  // namespace ax
