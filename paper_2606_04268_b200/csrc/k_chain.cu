// k_chain.cu — strategy CHAIN: every match of a FLATTENED stream in ONE streaming pass over the token stream that writes
// every output byte exactly once, coalesced, with no wave list, no atomics on the output and no zeroed output.
// After chain flattening no match reads bytes produced by another match of its own block (§3.3, invariant
// I3), so once the literal scatter has run, every match of block b depends on blocks < b only.  Tiles are taken in file
// order; a tile that holds a match of depth > 1 with a source before its block waits until every earlier block is
// completely written (a7: per-block completion counts instead of one grid barrier per depth —
// PAPER.md:224 "synchronization-bound"); dep[] is used only to skip the wait (dep == 1: all sources are literals).
// Per tile (512 sequences of one block, 256 threads, 3 CTAs per SM):
//   a2  the tile's cmd[] / len[] / dep[] / off[] slices and its slice of lit[] arrive in shared memory by 1-D bulk TMA
//       (cp.async.bulk + mbarrier), two stages: the tile after next is in flight; its descriptor is fetched by one thread
//       (cp.async) meanwhile
//   a3  scan inside the tile: thread t owns sequences 2t and 2t+1 through every phase (what it learns about them stays in
//       registers); warp shuffles + one barrier give every token's output position and literal offset (the tile's prefix
//       inside its block comes from k_tilesum)
//   a6  neighbouring lanes hold neighbouring tokens (neighbouring sources share L1 lines, neighbouring destinations share
//       image words):
//         before the wait  literal runs go into a shared-memory IMAGE of the tile's output span; each match is reduced to
//                          (aligned source address, destination, length / phase / period)
//         gather           the aligned 8-byte words holding each match's source travel global -> shared with cp.async
//                          (no registers held across the round trip; all of a thread's tokens in flight at once)
//         assemble         every match is written into the image with naturally aligned 1/2/4-byte stores (each byte has
//                          one owner: no merge, no zero fill), periodic if it overlaps its source (Q3); matches
//                          up to 32 bytes by one thread, longer ones by the whole warp
//       and the image goes to global memory with coalesced 16-byte vector stores (<= 15 head / tail bytes by byte stores;
//       measured against one bulk TMA store + its completion wait: 7.2 vs 7.7 ms on fastq1g — the wait is on the chain).
//       Tokens that would end beyond the image capacity (tiles with long matches / runs) are written straight to global
//       memory instead (their literal runs are there already: the literal scatter ran before).
// Rewriting a literal byte with its own value while another CTA reads it as a match source is harmless: a reader sees the
// old or the new copy of the same value.
#include "common.cuh"
#include "copy.cuh"

namespace ax {

constexpr int TILE = TILE_STREAM;                    // 512 sequences per tile
constexpr int SP_PER = 2;                            // tokens per thread (measured: 4 -> 2 cuts the hop from 10.3 to 8.1 us at 2048,
                                                     // and a 512-sequence tile spreads a block's ~370 tiles over all SMs: 7.1 us)
constexpr int SP_THREADS = TILE / SP_PER;            // 256
constexpr int SP_WARPS = SP_THREADS / 32;
constexpr int SP_OCC = 3;                            // CTAs per SM (77 registers per thread: measured 9.80 / 6.40 / 6.84 ms on fastq1g
                                                     // for 2 / 3 / 4 CTAs — at 4 the 64-register cap spills; at 2 less than one
                                                     // block's tiles are resident)
constexpr uint32_t SP_STRM = TILE * 10u;             // cmd | len | dep (2 B each) | off (4 B) per sequence
constexpr uint32_t SP_O_LEN = TILE * 2u, SP_O_DEP = TILE * 4u, SP_O_OFF = TILE * 6u;
constexpr uint32_t SP_IMG = 10 * TILE;               // image capacity in bytes (a text / FASTQ tile of 512 sequences spans ~3 KB)
constexpr uint32_t SP_LIT = 2 * TILE;                // staged slice of the block's lit[] (a text tile holds ~100 literal bytes)
constexpr uint32_t SP_SHORT = 16;                    // literal runs and self-overlapping matches up to this length: one thread
constexpr uint32_t SP_SHORT2 = 32;                   // other matches up to this length: one thread, two 16-byte pieces
static_assert(SP_THREADS % 32 == 0 && SP_THREADS <= 1024 && SP_THREADS * SP_PER == TILE, "one tile per CTA step");

// What one tile needs, gathered by the thread that issues its loads (while the previous tile is processed), so that the
// CTA does not walk tile_blk[] -> blocks[] -> tile_state[] (dependent global loads) on its critical path.
struct TileMeta {
    unsigned long long pre;                          // (out << 32 | lit) prefix of the tile inside its block
    const uint8_t* lit;                              // the block's lit[] in global memory
    uint32_t b, blk_lo, nt, prev_tiles;              // block, its first output byte, sequences in the tile, tiles of block b-1
    uint32_t lit16, lit_ok;                          // slit[0] = lit[lit16]; lit_ok: the tile's literal bytes are staged
};

// Descriptor of the NEXT tile, fetched by one thread straight into shared memory with cp.async (no registers held while
// it travels), in two steps so that the dependent loads (block descriptor after block index) are issued early and
// consumed late.
struct alignas(16) TileFetch {
    BlockDesc B;                                     // 64 bytes, 16-byte aligned in scratch
    unsigned long long pre, pre1;                    // tile_state[tile], tile_state[tile + 1]
    uint32_t b, prev_tiles, pad[2];                  // prev_tiles: tiles of block b-1 (0 for b = 0)
};
static_assert(sizeof(BlockDesc) == 64, "BlockDesc travels as four 16-byte cp.async");

struct SpanSmem {
    alignas(128) uint8_t strm[2][SP_STRM];           // two stages: the tile after next is in flight while this one is processed
    alignas(128) uint8_t slit[2][SP_LIT + 32];
    alignas(16) unsigned long long x0[TILE], x1[TILE], x2[TILE], x3[TILE], x4[TILE];   // the aligned words holding token j's source bytes
    alignas(128) uint8_t img[SP_IMG + 64];
    alignas(8) unsigned long long mbar[2];
    TileFetch fetch;                                 // (thread 0) descriptor of the next tile
    TileMeta meta[2];
    unsigned long long warp_sum[SP_WARPS];
    uint32_t img_end;                                // absolute end of the span held by the image
};

static_assert(sizeof(SpanSmem) + 1024 <= (228 * 1024) / SP_OCC, "SP_OCC CTAs (+1 KB reserved each) must fit the 228 KB of one SM");

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
__device__ __forceinline__ void cp_async8(void* smem, const void* gmem) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_u32(smem)), "l"(gmem) : "memory");
}

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(smem)), "l"(gmem) : "memory");
}
__device__ __forceinline__ void fetch_step1(const Params& P, TileFetch& F, uint32_t tile) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(smem_u32(&F.b)), "l"(P.tile_blk + tile) : "memory");
    cp_async8(&F.pre, P.tile_state + tile);
    if (tile + 1 < P.n_tiles) cp_async8(&F.pre1, P.tile_state + tile + 1);
    asm volatile("cp.async.commit_group;" ::: "memory");
}
__device__ __forceinline__ void fetch_step2(const Params& P, TileFetch& F) {
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    const uint8_t* src = reinterpret_cast<const uint8_t*>(P.blocks + F.b);
    uint8_t* dst = reinterpret_cast<uint8_t*>(&F.B);
#pragma unroll
    for (int i = 0; i < 4; ++i) cp_async16(dst + 16 * i, src + 16 * i);
    if (F.b) asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(smem_u32(&F.prev_tiles)), "l"(&P.blocks[F.b - 1].n_seq) : "memory");
    else F.prev_tiles = 0;                           // (holds n_seq of block b-1 until issue_tile_loads turns it into a tile count)
    asm volatile("cp.async.commit_group;" ::: "memory");
}

// The tile's stream slices (and its slice of lit[]) -> the stage, and its TileMeta (one elected thread).  Slices start on
// 4096-byte multiples of 16-byte aligned streams and are padded to 16 bytes inside the payload (docs/FORMAT.md), so sizes
// round up to 16 safely.  The arrive (release) orders the meta stores before any waiter's reads (acquire).
__device__ __forceinline__ void issue_tile_loads(const Params& P, SpanSmem& S, uint32_t tile, const TileFetch& F, uint32_t st) {
    const uint32_t j0 = (tile - F.B.tile_base) * TILE;
    const uint32_t left = F.B.n_seq - j0, n = left < (uint32_t)TILE ? left : (uint32_t)TILE;
    const uint32_t lit_lo = (uint32_t)F.pre, lit_hi = j0 + n < F.B.n_seq ? (uint32_t)F.pre1 : F.B.n_lit;
    const uint32_t l16 = lit_lo & ~15u;
    const uint32_t lbytes = lit_hi >= lit_lo ? (uint32_t)pad16(lit_hi) - l16 : 0xFFFFFFFFu;
    const bool lit_ok = lbytes <= SP_LIT;
    TileMeta& M = S.meta[st];
    M.pre = F.pre; M.lit = P.comp + F.B.lit_off; M.b = F.b; M.blk_lo = (uint32_t)F.B.out_base; M.nt = n;
    M.prev_tiles = (F.prev_tiles + TILE - 1) / TILE; M.lit16 = l16; M.lit_ok = lit_ok ? 1u : 0u;
    const uint32_t b2 = (uint32_t)pad16(2ull * n), b4 = (uint32_t)pad16(4ull * n);
    mbar_expect_tx(&S.mbar[st], 3 * b2 + b4 + (lit_ok ? lbytes : 0u));
    bulk_load(S.strm[st], P.comp + F.B.cmd_off + 2ull * j0, b2, &S.mbar[st]);
    bulk_load(S.strm[st] + SP_O_LEN, P.comp + F.B.len_off + 2ull * j0, b2, &S.mbar[st]);
    bulk_load(S.strm[st] + SP_O_DEP, P.comp + F.B.dep_off + 2ull * j0, b2, &S.mbar[st]);
    bulk_load(S.strm[st] + SP_O_OFF, P.comp + F.B.off_off + 4ull * j0, b4, &S.mbar[st]);
    if (lit_ok && lbytes) bulk_load(S.slit[st], P.comp + F.B.lit_off + l16, lbytes, &S.mbar[st]);
}
// bytes [sb, sb+16) of the 24-byte value (x0 | x1 << 64 | x2 << 128), sb in 0..7
__device__ __forceinline__ V16 extract16(unsigned long long x0, unsigned long long x1, unsigned long long x2, uint32_t sb) {
    const uint32_t s = sb * 8u;
    V16 v;
    if (s) { v.lo = (x0 >> s) | (x1 << (64u - s)); v.hi = (x1 >> s) | (x2 << (64u - s)); } else { v.lo = x0; v.hi = x1; }
    return v;
}

// chain_sync[32 + b] = finished tiles of block b.  It reaches the block's tile count only when blocks 0 .. b are ALL complete
// (words 0 .. 31 are unused padding: the counts start on their own 128-byte line)
constexpr uint32_t CH_CNT0 = 32;

__global__ void __launch_bounds__(SP_THREADS, SP_OCC) k_chain(Params P) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    SpanSmem& S = *reinterpret_cast<SpanSmem*>(smem_raw);
    const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    if (P.status->fault_flags != 0) return;          // a faulty stream is flagged, not decoded further (uniform: final before this launch)
    uint32_t tile = blockIdx.x;
    TileFetch& F = S.fetch;
    if (tid == 0) {
        mbar_init(&S.mbar[0], 1); mbar_init(&S.mbar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        for (uint32_t i = 0; i < 2u; ++i) {                               // the first two tiles of this CTA, one per stage
            const uint32_t t = tile + i * gridDim.x;
            if (t < P.n_tiles) {
                fetch_step1(P, F, t); fetch_step2(P, F);
                asm volatile("cp.async.wait_group 0;" ::: "memory");
                issue_tile_loads(P, S, t, F, i);
            }
        }
    }
    __syncthreads();
    uint32_t n_copied = 0;
    unsigned long long src_bytes = 0;                // M_src (this pass is the one that validates every match)

    for (uint32_t it = 0; tile < P.n_tiles; ++it, tile += gridDim.x) {
        const uint32_t st = it & 1u;
        const uint32_t next = tile + 2u * gridDim.x;                      // the tile that takes this stage over when this one is done
        const bool has_next = next < P.n_tiles;
        if (tid == 0 && has_next) fetch_step1(P, F, next);                 // consumed after the scan below
        // ---- a2: the tile's slices have landed (they were requested one tile ago)
        mbar_wait(&S.mbar[st], (it >> 1) & 1u);
        const TileMeta& M = S.meta[st];
        const unsigned long long pre = M.pre;
        const uint8_t* const lit = M.lit;
        const uint32_t b = M.b, blk_lo = M.blk_lo, nt = M.nt, prev_tiles = M.prev_tiles;
        const uint8_t* const lsrc_base = M.lit_ok ? S.slit[st] - M.lit16 : lit;   // byte x of the block's lit[] is lsrc_base[x]
        uint16_t* const s_cmd = reinterpret_cast<uint16_t*>(S.strm[st]);
        uint16_t* const s_len = reinterpret_cast<uint16_t*>(S.strm[st] + SP_O_LEN);
        uint16_t* const s_dep = reinterpret_cast<uint16_t*>(S.strm[st] + SP_O_DEP);
        uint32_t* const s_off = reinterpret_cast<uint32_t*>(S.strm[st] + SP_O_OFF);
        const uint32_t A0 = blk_lo + (uint32_t)(pre >> 32);               // absolute start of the tile's span
        const uint32_t img_org = A0 & ~15u;                               // absolute position of image byte 0
        // ================= before the wait (needs nothing another block wrote).  Thread t owns sequences 2t and 2t+1 through
        // every phase: what it learns about them stays in registers, and a token is only ever touched by its own thread.
        // ---- a3: scan of (cmd+len, cmd) packed as (hi, lo) of one u64
        const uint32_t jt = tid * SP_PER;
        uint32_t c[SP_PER], l[SP_PER], d[SP_PER], o[SP_PER];
        {
            uint32_t vc = 0, vl = 0, vd = 0; uint2 vo = make_uint2(0u, 0u);
            if (jt < nt) {
                vc = *reinterpret_cast<const uint32_t*>(s_cmd + jt); vl = *reinterpret_cast<const uint32_t*>(s_len + jt);
                vd = *reinterpret_cast<const uint32_t*>(s_dep + jt); vo = *reinterpret_cast<const uint2*>(s_off + jt);
            }
            c[0] = vc & 0xFFFFu; c[1] = vc >> 16; l[0] = vl & 0xFFFFu; l[1] = vl >> 16; d[0] = vd & 0xFFFFu; d[1] = vd >> 16;
            o[0] = vo.x; o[1] = vo.y;
            if (jt + 1u >= nt) { c[1] = 0; l[1] = 0; }                    // the tail shares its words with nothing: mask
        }
        unsigned long long tsum = 0;
        bool wait_src = false;                       // a match deeper than 1 reads an earlier block
#pragma unroll
        for (int k = 0; k < SP_PER; ++k) {
            tsum += ((unsigned long long)(c[k] + l[k]) << 32) | c[k];
            wait_src |= l[k] != 0 && o[k] < blk_lo && d[k] != 1u;
        }
        unsigned long long inc = tsum;
#pragma unroll
        for (int dd = 1; dd < 32; dd <<= 1) {
            const unsigned long long t = __shfl_up_sync(0xFFFFFFFFu, inc, dd);
            if (lane >= (uint32_t)dd) inc += t;
        }
        if (lane == 31) S.warp_sum[warp] = inc;
        if (tid == 0) S.img_end = A0;
        const bool must_wait = __syncthreads_or(wait_src) != 0;           // barrier 1
        unsigned long long wpre = 0;
#pragma unroll
        for (int w = 0; w < SP_WARPS; ++w) if (w < (int)warp) wpre += S.warp_sum[w];
        const unsigned long long ex = pre + wpre + (inc - tsum);
        // ---- token validation (I2, depth range, I3), literal runs into the image, every match reduced to what its copy needs:
        //   pp   destination            sa   source address (aligned down to 8 if one thread copies the match)
        //   inf  len (16 bits) | source byte phase (3) | period if the source overlaps, else 0 (4) | in image | by one thread
        uint32_t pp[SP_PER], sa[SP_PER], inf[SP_PER], ps[SP_PER], lp[SP_PER];
        {
            uint32_t p = blk_lo + (uint32_t)(ex >> 32), ls = (uint32_t)ex, fit_end = 0;
            bool bad_src = false, bad_dep = false, long_lit = false;
#pragma unroll
            for (int k = 0; k < SP_PER; ++k) {
                ps[k] = p; lp[k] = ls;
                const uint32_t mdst = p + c[k], len = l[k];
                const bool in_img = mdst + len - img_org <= SP_IMG;       // tokens are monotone: a prefix of the tile fits the image
                pp[k] = mdst; inf[k] = in_img ? 1u << 23 : 0u; sa[k] = 0;
                if (len) {
                    if (o[k] >= mdst || len < P.min_match) bad_src = true;
                    else if (d[k] == 0 || d[k] > P.max_depth || (o[k] >= blk_lo && d[k] != 1u)) bad_dep = true;   // (in-block source: literal only)
                    else {
                        const uint32_t dist = mdst - o[k];
                        const bool ovl = dist < len;
                        const bool by_thread = len <= SP_SHORT || (len <= SP_SHORT2 && !ovl);
                        sa[k] = by_thread ? (o[k] & ~7u) : o[k];
                        inf[k] |= len | (o[k] & 7u) << 16 | (ovl && by_thread ? dist : 0u) << 19 | (by_thread ? 1u << 26 : 0u);
                        ++n_copied; src_bytes += ovl ? dist : len;
                    }
                }
                if (c[k] && in_img) {
                    if (c[k] <= SP_SHORT) place16(S.img + (p - img_org), load16(lsrc_base + ls, c[k]), c[k]);
                    else long_lit = true;
                }
                p = mdst + len;
                ls += c[k];
                if (in_img) fit_end = p;
            }
            if (bad_src) raise_fault(P.status, F_SOURCE, b);              // a faulty match is flagged and skipped: its bytes stay a hole
            if (bad_dep) raise_fault(P.status, F_DEPTH, b);
            fit_end = __reduce_max_sync(0xFFFFFFFFu, fit_end);
            if (lane == 0 && fit_end) atomicMax(&S.img_end, fit_end);
            if (__any_sync(0xFFFFFFFFu, long_lit)) {                      // long literal runs: the whole warp copies each
#pragma unroll
                for (int k = 0; k < SP_PER; ++k) {
                    uint32_t m = __ballot_sync(0xFFFFFFFFu, c[k] > SP_SHORT && ((inf[k] >> 23) & 1u));
                    while (m) {
                        const int sl = __ffs(m) - 1; m &= m - 1;
                        const uint32_t d2 = __shfl_sync(0xFFFFFFFFu, ps[k], sl), s2 = __shfl_sync(0xFFFFFFFFu, lp[k], sl), n2 = __shfl_sync(0xFFFFFFFFu, c[k], sl);
                        warp_copy(S.img + (d2 - img_org), lit + s2, n2, lane);
                    }
                }
            }
        }
        if (tid == 0 && has_next) fetch_step2(P, F);                       // (its block index has arrived by now)
        if (must_wait && b) {
            // a7: every block before this one completely written?  count[b-1] reaches the tile count of block b-1 only when
            // blocks 0 .. b-1 are all complete (a tile publishes only after it has seen block b-2's count complete: here, or
            // before its publish below), so this one word is the whole condition.  One thread spins; the poll itself is the
            // acquire (SASS: LDG.STRONG.GPU + CCTL.IVALL, which also drops this SM's L1 so that the gathers below see what
            // other SMs wrote): a relaxed poll followed by fence.acq_rel.gpu puts a MEMBAR.ALL.GPU in front of the gathers
            // (measured 6.70 vs 6.39 ms per decode on fastq1g).
            if (tid == 0) {
                uint32_t v;
                for (;;) {
                    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(P.chain_sync + CH_CNT0 + b - 1u) : "memory");
                    if (v >= prev_tiles) break;
                    if (v == 0) __nanosleep(400);                         // block b-1 has not begun to finish: keep the hot line's queue short
                }
            }
            __syncthreads();                                              // barrier 2
        }
        // ================= after the wait.  Gather: the aligned 8-byte words holding each match's source travel global ->
        // shared (cp.async: no registers held across the round trip, both tokens of the thread in flight at once)
#pragma unroll
        for (int k = 0; k < SP_PER; ++k) {
            if (!((inf[k] >> 26) & 1u)) continue;
            const uint32_t j = k * SP_THREADS + tid;                       // the thread's private slot
            const uint32_t per = (inf[k] >> 19) & 15u;
            const uint32_t span = ((inf[k] >> 16) & 7u) + (per ? per : (inf[k] & 0xFFFFu));
            const uint8_t* g = P.out + sa[k];
            cp_async8(&S.x0[j], g);
            if (span > 8u) cp_async8(&S.x1[j], g + 8);
            if (span > 16u) cp_async8(&S.x2[j], g + 16);
            if (span > 24u) cp_async8(&S.x3[j], g + 24);
            if (span > 32u) cp_async8(&S.x4[j], g + 32);
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
        asm volatile("cp.async.wait_group 0;" ::: "memory");
        // ---- a6: every match into the image (or, beyond its capacity, straight to global memory)
        bool any_long = false;
#pragma unroll
        for (int k = 0; k < SP_PER; ++k) {
            const uint32_t ll = inf[k] & 0xFFFFu;
            any_long |= ll != 0 && !((inf[k] >> 26) & 1u);
            if ((inf[k] >> 26) & 1u) {
                const uint32_t j = k * SP_THREADS + tid, per = (inf[k] >> 19) & 15u, sb = (inf[k] >> 16) & 7u;
                const unsigned long long y2 = S.x2[j];
                V16 v = extract16(S.x0[j], S.x1[j], y2, sb);
                if (per) v = extend_period(v, per);                        // self-overlap: periodic extension (Q3)
                const uint32_t l0 = ll < 16u ? ll : 16u;
                if ((inf[k] >> 23) & 1u) {
                    place16(S.img + (pp[k] - img_org), v, l0);
                    if (ll > 16u) place16(S.img + (pp[k] - img_org) + 16, extract16(y2, S.x3[j], S.x4[j], sb), ll - 16u);
                } else {
                    store16(P.out + pp[k], v, l0);
                    if (ll > 16u) store16(P.out + pp[k] + 16, extract16(y2, S.x3[j], S.x4[j], sb), ll - 16u);
                }
            }
        }
        if (__any_sync(0xFFFFFFFFu, any_long)) {                          // long matches: the whole warp copies each
#pragma unroll
            for (int k = 0; k < SP_PER; ++k) {
                uint32_t m = __ballot_sync(0xFFFFFFFFu, (inf[k] & 0xFFFFu) != 0 && !((inf[k] >> 26) & 1u));
                while (m) {
                    const int sl = __ffs(m) - 1; m &= m - 1;
                    const uint32_t d2 = __shfl_sync(0xFFFFFFFFu, pp[k], sl), o2 = __shfl_sync(0xFFFFFFFFu, sa[k], sl), f2 = __shfl_sync(0xFFFFFFFFu, inf[k], sl);
                    const bool im2 = (f2 >> 23) & 1u;
                    uint8_t* dst = im2 ? S.img + (d2 - img_org) : P.out + d2;
                    warp_match(dst, P.out + o2, f2 & 0xFFFFu, d2 - o2, !im2, lane);
                }
            }
        }
        __syncthreads();                                                  // barrier 4: image complete, stage free
        {
            // ---- write the image out: 16-byte chunks by plain coalesced vector stores, the partial chunks at both ends by bytes
            const uint32_t E = S.img_end;
            const uint32_t c0 = (A0 + 15u) & ~15u, c1 = E & ~15u;
            if (c1 > c0) {
                const uint4* src = reinterpret_cast<const uint4*>(S.img + (c0 - img_org));
                uint4* dst = reinterpret_cast<uint4*>(P.out + c0);
                for (uint32_t i = tid; i < ((c1 - c0) >> 4); i += SP_THREADS) dst[i] = src[i];
            }
            if (tid == 0 && has_next) issue_tile_loads(P, S, next, F, st);   // the stage is free
            const uint32_t he = c0 < E ? c0 : E;                          // head bytes [A0, he)
            if (tid >= 32u && tid < 48u && A0 + (tid - 32u) < he) P.out[A0 + (tid - 32u)] = S.img[A0 + (tid - 32u) - img_org];
            if (tid >= 48u && tid < 64u && c1 >= c0) {                    // tail bytes [c1, E)
                const uint32_t a = c1 + (tid - 48u);
                if (a < E) P.out[a] = S.img[a - img_org];
            }
            __syncthreads();                                              // barrier 5: every store of the tile is issued
            if (tid == 0) {
                // publish.  A tile that did not have to wait still may not count before blocks < b are complete (see the
                // wait above: count[b] complete must imply that); it has normally long been the case.
                if (!must_wait && b) {
                    uint32_t v;
                    do { asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(P.chain_sync + CH_CNT0 + b - 1u) : "memory"); } while (v < prev_tiles);
                }
                asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(P.chain_sync + CH_CNT0 + b), "r"(1u) : "memory");
            }
        }
    }
#pragma unroll
    for (int d = 16; d; d >>= 1) n_copied += __shfl_xor_sync(0xFFFFFFFFu, n_copied, d);
    if (lane == 0 && n_copied) atomicAdd(&P.status->n_final, n_copied);
    {
#pragma unroll
        for (int d = 16; d; d >>= 1) src_bytes += __shfl_xor_sync(0xFFFFFFFFu, src_bytes, d);
        if (lane == 0 && src_bytes) atomicAdd(&P.status->match_src_bytes, src_bytes);
    }
}

cudaError_t chain_configure() {
    return cudaFuncSetAttribute(k_chain, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(SpanSmem));
}

int chain_max_ctas_per_sm() {
    int n = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k_chain, SP_THREADS, sizeof(SpanSmem)) != cudaSuccess) return 0;
    return n;
}

// Every tile of the grid must be resident (a tile spins until lower tiles are done), so the launch is cooperative and the
// grid at most n_sm x occupancy; the per-block counts start from zero.
cudaError_t launch_chain(const Params& P, int grid, cudaStream_t st) {
    if (!P.n_tiles) return cudaSuccess;
    cudaError_t e = cudaMemsetAsync(P.chain_sync, 0, sizeof(uint32_t) * (CH_CNT0 + (size_t)P.n_blocks), st);
    if (e != cudaSuccess) return e;
    const uint32_t g = (uint32_t)grid < P.n_tiles ? grid : P.n_tiles;
    Params p = P;
    void* args[] = {&p};
    return cudaLaunchCooperativeKernel((const void*)k_chain, dim3(g), dim3(SP_THREADS), args, sizeof(SpanSmem), st);
}

size_t chain_sync_words(uint32_t n_blocks) { return CH_CNT0 + (size_t)n_blocks; }

}  // namespace ax
