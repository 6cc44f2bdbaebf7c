// k_tilesum.cu — step a3, block level: the exclusive prefix of (cmd+len, cmd) of every tile inside its block, i.e. the
// sequential walk of PAPER.md:53 ("processes cmd[] in sequence") restated as a two-level scan: this kernel produces one
// prefix per tile (Params::tile sequences), the consumers (k_pre, k_pass, k_chain) scan inside the tile with warp shuffles.  Also writes
// the tile -> block map and checks invariant I1 (the block's tokens sum to raw_len, its literal runs to n_lit): every
// later kernel relies on it — with the totals right, every token's range lies inside its block.
// One CTA per 1 MB block; each WARP sums whole tiles on its own (all its loads independent), then one
// warp scans the tile totals.  Blocks with more than TS_CHUNK tiles are walked in chunks with a carry.
#include "common.cuh"

namespace ax {

constexpr int TS_THREADS = 256;
constexpr int TS_WARPS = TS_THREADS / 32;
constexpr uint32_t TS_CHUNK = 1024;

__global__ void __launch_bounds__(TS_THREADS) k_tilesum(Params P) {
    __shared__ unsigned long long s_tot[TS_CHUNK];
    __shared__ unsigned long long s_carry;
    if (P.status->fault_flags & F_INDEX) return;         // the block index itself is inconsistent: nothing below is safe
    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    for (uint32_t b = blockIdx.x; b < P.n_blocks; b += gridDim.x) {
        const BlockDesc B = P.blocks[b];
        const uint32_t nt = (B.n_seq + P.tile - 1) / P.tile;
        __syncthreads();
        if (tid == 0) s_carry = 0;
        for (uint32_t t0 = 0; t0 < nt; t0 += TS_CHUNK) {
            const uint32_t tn = nt - t0 < TS_CHUNK ? nt - t0 : TS_CHUNK;
            for (uint32_t t = warp; t < tn; t += TS_WARPS) {
                unsigned long long s = 0;
                for (uint32_t r = 0; r < P.tile / 256; ++r) {                // (tile is a multiple of 256)
                    const uint32_t j0 = (t0 + t) * P.tile + r * 256 + lane * 8;
                    if (j0 < B.n_seq) {
                        const uint4 vc = *reinterpret_cast<const uint4*>(P.comp + B.cmd_off + 2ull * j0);
                        const uint4 vl = *reinterpret_cast<const uint4*>(P.comp + B.len_off + 2ull * j0);
                        uint32_t c[8], l[8];
                        unpack8(vc, c); unpack8(vl, l);
#pragma unroll
                        for (int k = 0; k < 8; ++k)
                            if (j0 + k < B.n_seq) s += ((unsigned long long)(c[k] + l[k]) << 32) | c[k];
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
                    if (i < tn) { P.tile_state[B.tile_base + t0 + i] = ex; P.tile_blk[B.tile_base + t0 + i] = b; }
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

void launch_tilesum(const Params& P, int grid, cudaStream_t st) {
    if (P.n_blocks) k_tilesum<<<(uint32_t)grid < P.n_blocks ? grid : P.n_blocks, TS_THREADS, 0, st>>>(P);
}

}  // namespace ax
