// k_span.cu — strategy SPAN, the last match wave of a shallow stream (e.g. the depth-limited encoder of PAPER.md:228
// §7.4, where the depth limit piles most matches up at depth D) as ONE streaming pass over the token stream that
// writes every output byte exactly once, coalesced, with no wave list, no atomics and no zeroed output:
//   a2  parse: the tile's cmd[] / len[] / dep[] / off[] slices arrive in shared memory by 1-D bulk TMA
//       (cp.async.bulk + mbarrier), double-buffered: the next tile's 20 KB are in flight while this one is copied
//   a3  scan inside the tile (warp shuffles); the tile's prefix inside its block comes from k_tilesum
//   a6  every token of the tile is materialised into a shared-memory IMAGE of the tile's output span:
//         literal run              <- lit[]
//         match with dep == D      <- out[off ..)   (its sources were written by the earlier waves)
//         match with dep <  D      <- out[mdst ..)  (its own bytes, already written by its wave)
//       then the image goes to global memory with one bulk TMA store (16-byte chunks; <= 15 head / tail bytes by
//       byte stores).  Each thread owns 8 consecutive sequences, i.e. one contiguous piece of the span, and assembles it
//       with a register byte-stream writer: whole 8-byte words go to the image with plain shared-memory stores, the
//       partial word at each thread boundary travels to its neighbour by shuffle (no shared-memory atomics).
// Threads whose piece would end beyond the image capacity (tiles with long matches / runs) write their depth-D matches
// straight to global memory instead (everything else of theirs is there already).
// Rewriting a byte of depth < D with its own value while another CTA reads it as a match source is harmless: a
// reader sees the old or the new copy of the same value.
#include "common.cuh"
#include "copy.cuh"

namespace ax {

constexpr int SP_THREADS = PRE_THREADS;              // 256 threads x 8 sequences = one tile per CTA step
constexpr int SP_WARPS = SP_THREADS / 32;
constexpr uint32_t SP_STRM = TILE * 10u;             // cmd | len | dep (2 B each) | off (4 B) per sequence
constexpr uint32_t SP_O_LEN = TILE * 2u, SP_O_DEP = TILE * 4u, SP_O_OFF = TILE * 6u;
#ifndef AX_SP_IMG
#define AX_SP_IMG (28 * 1024)
#endif
constexpr uint32_t SP_IMG = AX_SP_IMG;               // image capacity in bytes (a text / FASTQ tile spans ~12 KB)
constexpr uint32_t KEY_NONE = 0xFFFFFFFFu;
#ifndef AX_SP_OCC
#define AX_SP_OCC 2
#endif

struct SpanSmem {
    alignas(128) uint8_t strm[2][SP_STRM];
    alignas(128) uint8_t img[SP_IMG + 64];
    alignas(8) unsigned long long mbar[2];
    unsigned long long warp_sum[SP_WARPS];
    unsigned long long tail_val[SP_WARPS];           // per warp: lane 31's chained partial word ...
    uint32_t tail_key[SP_WARPS];                     // ... the image word it belongs to ...
    uint32_t head_key[SP_WARPS];                     // ... and the first image word of the warp's lane 0
    uint32_t n_img[SP_WARPS];                        // image-mode threads per warp
    uint32_t img_end[2];                             // absolute end of the span held by the image (slot = iteration parity)
};

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(unsigned long long* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, uint32_t parity) {
    uint32_t ok;
    do {
        asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}"
                     : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    } while (!ok);
}
// 1-D bulk TMA: global -> shared, completion counted in bytes on an mbarrier (SASS: UBLKCP)
__device__ __forceinline__ void bulk_load(void* smem, const void* gmem, uint32_t bytes, unsigned long long* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(smem)), "l"(gmem), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
// 1-D bulk TMA: shared -> global, tracked by the thread's bulk async-group
__device__ __forceinline__ void bulk_store(void* gmem, const void* smem, uint32_t bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(gmem), "r"(smem_u32(smem)), "r"(bytes) : "memory");
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
}

// The tile's four stream slices -> stage `st` (one elected thread).  Slices start on 4096-byte multiples of 16-byte
// aligned streams and are padded to 16 bytes inside the payload (docs/FORMAT.md), so sizes round up to 16 safely.
__device__ __forceinline__ void issue_tile_loads(const Params& P, SpanSmem& S, uint32_t tile, uint32_t st) {
    const uint32_t b = P.tile_blk[tile];
    const BlockDesc* B = P.blocks + b;
    const uint32_t j0 = (tile - B->tile_base) * TILE;
    const uint32_t left = B->n_seq - j0, n = left < (uint32_t)TILE ? left : (uint32_t)TILE;
    const uint32_t b2 = (uint32_t)pad16(2ull * n), b4 = (uint32_t)pad16(4ull * n);
    mbar_expect_tx(&S.mbar[st], 3 * b2 + b4);
    bulk_load(S.strm[st], P.comp + B->cmd_off + 2ull * j0, b2, &S.mbar[st]);
    bulk_load(S.strm[st] + SP_O_LEN, P.comp + B->len_off + 2ull * j0, b2, &S.mbar[st]);
    bulk_load(S.strm[st] + SP_O_DEP, P.comp + B->dep_off + 2ull * j0, b2, &S.mbar[st]);
    bulk_load(S.strm[st] + SP_O_OFF, P.comp + B->off_off + 4ull * j0, b4, &S.mbar[st]);
}

// ---- register byte-stream writer: appends byte strings to the contiguous piece [start, ..) of the image.
// Whole words are stored as they fill up, except the thread's FIRST word, which is kept in `first` until the partial
// word of the preceding thread has been merged in (finish protocol in the kernel).
struct SpanWriter {
    unsigned long long acc, first;
    unsigned long long* img;
    uint32_t nfill, w, fw;                           // bytes used in acc; image word acc belongs to; first word of the thread
    __device__ __forceinline__ void init(unsigned long long* img_, uint32_t rel) {
        img = img_; w = rel >> 3; fw = w; nfill = rel & 7u; acc = 0ull; first = 0ull;
    }
    __device__ __forceinline__ void emit(unsigned long long x) {
        if (w == fw) first = x; else img[w] = x;
        ++w;
    }
    // v: n (1..16) valid bytes, everything above them zero
    __device__ __forceinline__ void append(V16 v, uint32_t n) {
        const uint32_t sh = nfill * 8u, tot = nfill + n;
        unsigned long long w0 = v.lo, c1 = v.hi, c2 = 0ull;
        if (sh) { w0 = acc | (v.lo << sh); c1 = (v.lo >> (64u - sh)) | (v.hi << sh); c2 = v.hi >> (64u - sh); }
        if (tot >= 8u) {
            emit(w0);
            if (tot >= 16u) { emit(c1); acc = c2; } else acc = c1;
        } else acc = w0;
        nfill = tot & 7u;
    }
    // n bytes that somebody else writes (a long token, copied later by the whole warp): zeros for now
    __device__ __forceinline__ void skip(uint32_t n) {
        const uint32_t tot = nfill + n;
        if (tot >= 8u) { emit(acc); w += (tot >> 3) - 1u; acc = 0ull; }
        nfill = tot & 7u;
    }
};

__device__ __forceinline__ V16 mask_bytes(V16 v, uint32_t n) {                  // keep the first n (1..16) bytes
    if (n < 8u) { v.lo &= (1ull << (n * 8u)) - 1ull; v.hi = 0ull; }
    else if (n < 16u) v.hi &= n == 8u ? 0ull : (1ull << ((n - 8u) * 8u)) - 1ull;
    return v;
}

// bytes [sb, sb+16) of the 32-byte pair (wa | wb << 128), sb in 0..15
__device__ __forceinline__ V16 extract16(uint4 wa, uint4 wb, uint32_t sb) {
    const unsigned long long a0 = (unsigned long long)wa.x | ((unsigned long long)wa.y << 32), a1 = (unsigned long long)wa.z | ((unsigned long long)wa.w << 32),
                             b0 = (unsigned long long)wb.x | ((unsigned long long)wb.y << 32), b1 = (unsigned long long)wb.z | ((unsigned long long)wb.w << 32);
    const unsigned long long x0 = sb < 8u ? a0 : a1, x1 = sb < 8u ? a1 : b0, x2 = sb < 8u ? b0 : b1;
    const uint32_t s = (sb & 7u) * 8u;
    V16 v;
    if (s) { v.lo = (x0 >> s) | (x1 << (64u - s)); v.hi = (x1 >> s) | (x2 << (64u - s)); } else { v.lo = x0; v.hi = x1; }
    return v;
}

constexpr uint32_t SP_SHORT = 16;                    // tokens up to this length go through the thread's registers

__global__ void __launch_bounds__(SP_THREADS, AX_SP_OCC) k_span(Params P, uint32_t depth_hi) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    SpanSmem& S = *reinterpret_cast<SpanSmem*>(smem_raw);
    const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    if (P.status->fault_flags != 0) return;          // a faulty stream is flagged, not decoded further (uniform: final before this launch)
    if (tid == 0) {
        mbar_init(&S.mbar[0], 1); mbar_init(&S.mbar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    uint32_t tile = blockIdx.x;
    if (tid == 0 && tile < P.n_tiles) issue_tile_loads(P, S, tile, 0);
    uint32_t n_copied = 0;
    unsigned long long* const img64 = reinterpret_cast<unsigned long long*>(S.img);

    for (uint32_t it = 0; tile < P.n_tiles; ++it, tile += gridDim.x) {
        const uint32_t st = it & 1u, par = (it >> 1) & 1u;
        // stage st^1 was last read in iteration it-1, and every thread has passed a __syncthreads since
        if (tid == 0 && tile + gridDim.x < P.n_tiles) issue_tile_loads(P, S, tile + gridDim.x, st ^ 1u);
        const uint32_t b = P.tile_blk[tile];
        const unsigned long long pre = P.tile_state[tile];
        const BlockDesc* B = P.blocks + b;
        const uint32_t blk_lo = (uint32_t)B->out_base, tile_base = B->tile_base, n_seq = B->n_seq;
        const uint8_t* lit = P.comp + B->lit_off;
        const uint32_t j0 = (tile - tile_base) * TILE, left = n_seq - j0, nt = left < (uint32_t)TILE ? left : (uint32_t)TILE;
        const uint32_t jt = tid * PRE_ITEMS;
        // ---- a2: parse from the staged slices
        mbar_wait(&S.mbar[st], par);
        Seq8 q;
        {
            const uint8_t* sb = S.strm[st];
            const uint4 z = make_uint4(0u, 0u, 0u, 0u);
            if (jt < nt)
                parse8(q, *reinterpret_cast<const uint4*>(sb + 2u * jt), *reinterpret_cast<const uint4*>(sb + SP_O_LEN + 2u * jt),
                       *reinterpret_cast<const uint4*>(sb + SP_O_DEP + 2u * jt), *reinterpret_cast<const uint4*>(sb + SP_O_OFF + 4u * jt),
                       *reinterpret_cast<const uint4*>(sb + SP_O_OFF + 4u * jt + 16u), nt - jt);
            else parse8(q, z, z, z, z, z, 0);
        }
        // ---- a3: scan of (cmd+len, cmd) packed as (hi, lo) of one u64
        unsigned long long tsum = 0;
#pragma unroll
        for (int k = 0; k < PRE_ITEMS; ++k) tsum += ((unsigned long long)(q.c[k] + q.l[k]) << 32) | q.c[k];
        unsigned long long inc = tsum;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const unsigned long long t = __shfl_up_sync(0xFFFFFFFFu, inc, d);
            if (lane >= (uint32_t)d) inc += t;
        }
        if (lane == 31) S.warp_sum[warp] = inc;
        const uint32_t A0 = blk_lo + (uint32_t)(pre >> 32);               // absolute start of the tile's span
        const uint32_t img_org = A0 & ~15u;                               // absolute position of image byte 0
        if (tid == 0) {
            asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");   // the previous tile's store has read the image
            S.img_end[st] = A0;
        }
        __syncthreads();
        unsigned long long wpre = 0;
#pragma unroll
        for (int w = 0; w < SP_WARPS; ++w) if (w < (int)warp) wpre += S.warp_sum[w];
        const unsigned long long ex = pre + wpre + (inc - tsum);
        const uint32_t ts = blk_lo + (uint32_t)(ex >> 32);                // absolute start of this thread's piece
        const uint32_t te = ts + (uint32_t)(tsum >> 32);
        const uint32_t lsrc0 = (uint32_t)ex;                              // offset inside the block's lit[]
        const bool use_img = te - img_org <= SP_IMG;                      // a prefix of the CTA's threads (te is monotone)
        {
            const uint32_t m = __reduce_max_sync(0xFFFFFFFFu, use_img ? te : 0u);
            const uint32_t cnt = __popc(__ballot_sync(0xFFFFFFFFu, use_img));
            if (lane == 0) { if (cnt) atomicMax(&S.img_end[st], m); S.n_img[warp] = cnt; }
        }
        SpanWriter W;
        W.init(img64, ts - img_org);
        uint32_t p = ts, ls = lsrc0;
        uint32_t bad = 0;                                                 // bit k: match k is invalid (hole)
        bool has_long = false;
        // ---- a6: two batches of four tokens: all gathers of a batch are issued before the first append
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            uint4 wa[4], wb[4];
            uint32_t pp = p;
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const int k = 4 * h + i;
                pp += q.c[k];
                const uint32_t l = q.l[k];
                wa[i] = make_uint4(0u, 0u, 0u, 0u); wb[i] = wa[i];
                if (l) {
                    const bool deep = q.dp[k] == depth_hi;
                    if (q.of[k] >= pp || q.dp[k] == 0 || q.dp[k] > depth_hi) bad |= 1u << k;
                    else if (l <= SP_SHORT && (use_img || deep)) {
                        const uint32_t src = deep ? q.of[k] : pp;
                        const uint32_t dist = pp - q.of[k];
                        const uint32_t need = (deep && dist < l) ? dist : l;
                        const uint4* g = reinterpret_cast<const uint4*>(P.out + (src & ~15u));
                        wa[i] = g[0];
                        if ((src & 15u) + need > 16u) wb[i] = g[1];
                    }
                }
                pp += l;
            }
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const int k = 4 * h + i;
                const uint32_t c = q.c[k], l = q.l[k];
                if (c) {                                                  // literal run (rare on compressible data)
                    if (use_img) {
                        if (c <= SP_SHORT) W.append(mask_bytes(load16(lit + ls, c), c), c);
                        else { W.skip(c); has_long = true; }
                    }
                    p += c; ls += c;
                }
                if (l) {
                    const bool deep = q.dp[k] == depth_hi, ok = !(bad & (1u << k));
                    if (ok && deep) ++n_copied;
                    if (l <= SP_SHORT && ok && (use_img || deep)) {
                        const uint32_t src = deep ? q.of[k] : p, dist = p - q.of[k];
                        V16 v = extract16(wa[i], wb[i], src & 15u);
                        if (deep && dist < l) v = extend_period(v, dist);  // self-overlap: periodic extension (Q3)
                        v = mask_bytes(v, l);
                        if (use_img) W.append(v, l); else store16(P.out + p, v, l);
                    } else {
                        if (use_img) W.skip(l);
                        if (ok && (use_img || deep)) has_long = true;
                    }
                    p += l;
                }
            }
        }
        if (bad) raise_fault(P.status, F_SOURCE, b);
        // ---- finish protocol: the partial last word of every piece is merged into the first word of the next piece
        // (segmented OR-scan keyed by image word: pieces shorter than a word chain through several lanes)
        unsigned long long val = use_img ? W.acc : 0ull;
        const uint32_t key = use_img ? W.w : KEY_NONE;
        const bool tiny = use_img && W.w == W.fw;                         // the piece never left its first word
        if (__any_sync(0xFFFFFFFFu, tiny)) {
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const unsigned long long v2 = __shfl_up_sync(0xFFFFFFFFu, val, d);
                const uint32_t k2 = __shfl_up_sync(0xFFFFFFFFu, key, d);
                if (lane >= (uint32_t)d && k2 == key) val |= v2;
            }
        }
        if (lane == 31) { S.tail_val[warp] = val; S.tail_key[warp] = key; }
        if (lane == 0) S.head_key[warp] = use_img ? W.fw : KEY_NONE;
        const bool any_long = __syncthreads_or(has_long);                 // barrier A
        {
            // what the preceding warps contribute to this warp's first word fw0: the tail of warp-1, and of the warps
            // before it for as long as a whole warp lies inside that one word
            const uint32_t fw0 = __shfl_sync(0xFFFFFFFFu, use_img ? W.fw : KEY_NONE, 0);
            unsigned long long carry = 0ull;
            if (lane == 0 && use_img) {
                for (int j = (int)warp - 1; j >= 0; --j) {
                    if (S.tail_key[j] != fw0) break;
                    carry |= S.tail_val[j];
                    if (S.head_key[j] != S.tail_key[j]) break;
                }
            }
            carry = __shfl_sync(0xFFFFFFFFu, carry, 0);
            if (use_img && key == fw0) val |= carry;                      // lanes whose chain reaches back past lane 0
            const unsigned long long prev = __shfl_up_sync(0xFFFFFFFFu, val, 1);
            const unsigned long long chain_in = lane ? prev : carry;      // the preceding piece ends where this one starts
            uint32_t n_img = 0;
#pragma unroll
            for (int w = 0; w < SP_WARPS; ++w) n_img += S.n_img[w];
            if (use_img && !tiny) img64[W.fw] = W.first | chain_in;
            if (use_img && tid + 1 == n_img) img64[key] = val;            // last image piece: its (chained) partial word
        }
        // ---- long tokens: the whole warp copies each (image mode: into the image; direct mode: depth-D matches only)
        if (any_long) {
            __syncthreads();                                              // barrier B: short stores before long copies into the same words
            uint32_t p2 = ts, ls2 = lsrc0;
#pragma unroll
            for (int k = 0; k < PRE_ITEMS; ++k) {
                const uint32_t c = q.c[k], l = q.l[k];
                uint32_t m = __ballot_sync(0xFFFFFFFFu, use_img && c > SP_SHORT);
                while (m) {
                    const int sl = __ffs(m) - 1; m &= m - 1;
                    const uint32_t d2 = __shfl_sync(0xFFFFFFFFu, p2, sl), s2 = __shfl_sync(0xFFFFFFFFu, ls2, sl), n2 = __shfl_sync(0xFFFFFFFFu, c, sl);
                    warp_copy(S.img + (d2 - img_org), lit + s2, n2, lane);
                }
                p2 += c; ls2 += c;
                const bool deep = q.dp[k] == depth_hi;
                m = __ballot_sync(0xFFFFFFFFu, l > SP_SHORT && !(bad & (1u << k)) && (use_img || deep));
                while (m) {
                    const int sl = __ffs(m) - 1; m &= m - 1;
                    const uint32_t d2 = __shfl_sync(0xFFFFFFFFu, p2, sl), o2 = __shfl_sync(0xFFFFFFFFu, q.of[k], sl), n2 = __shfl_sync(0xFFFFFFFFu, l, sl);
                    const bool dp2 = __shfl_sync(0xFFFFFFFFu, (uint32_t)deep, sl) != 0, im2 = __shfl_sync(0xFFFFFFFFu, (uint32_t)use_img, sl) != 0;
                    uint8_t* dst = im2 ? S.img + (d2 - img_org) : P.out + d2;
                    if (dp2) warp_match(dst, P.out + o2, n2, d2 - o2, false, lane);
                    else warp_copy(dst, P.out + d2, n2, lane);              // (image mode only) its own bytes
                }
                p2 += l;
            }
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");      // generic-proxy image writes -> visible to the bulk store
        __syncthreads();                                                  // barrier C
        // ---- write the image out: 16-byte chunks by one bulk TMA store, the partial chunks at both ends by byte stores
        {
            const uint32_t E = S.img_end[st];
            const uint32_t c0 = (A0 + 15u) & ~15u, c1 = E & ~15u;
            if (tid == 0 && c1 > c0) bulk_store(P.out + c0, S.img + (c0 - img_org), c1 - c0);
            const uint32_t he = c0 < E ? c0 : E;                          // head bytes [A0, he)
            if (tid < 16u && A0 + tid < he) P.out[A0 + tid] = S.img[A0 + tid - img_org];
            if (tid >= 16u && tid < 32u && c1 >= c0) {                    // tail bytes [c1, E)
                const uint32_t a = c1 + (tid - 16u);
                if (a < E) P.out[a] = S.img[a - img_org];
            }
        }
    }
    if (tid == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
#pragma unroll
    for (int d = 16; d; d >>= 1) n_copied += __shfl_xor_sync(0xFFFFFFFFu, n_copied, d);
    if (lane == 0 && n_copied) atomicAdd(&P.status->n_final, n_copied);
}

size_t span_smem_bytes() { return sizeof(SpanSmem); }

cudaError_t span_configure() {
    return cudaFuncSetAttribute(k_span, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(SpanSmem));
}

int span_max_ctas_per_sm() {
    int n = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k_span, SP_THREADS, sizeof(SpanSmem)) != cudaSuccess) return 0;
    return n;
}

void launch_span(const Params& P, uint32_t depth_hi, int grid, cudaStream_t st) {
    if (!P.n_tiles) return;
    const uint32_t g = (uint32_t)grid < P.n_tiles ? grid : P.n_tiles;
    k_span<<<g, SP_THREADS, sizeof(SpanSmem), st>>>(P, depth_hi);
}

}  // namespace ax
