// copy.cuh — byte-copy primitives of the match copy (step a6) shared by the wave kernel (k_match.cu) and the fused
// tile kernel (k_fused.cu).  All take explicit destination / source pointers (generic: global or shared memory).
// Contract of every routine: it stores exactly the bytes [d, d+len) and nothing else; it loads only from
// [s - 15, s + min(len, dist) + 15] rounded to aligned words — never a byte the match itself produces, unless the
// routine says so (warp_match's doubling, which requires source and destination to live in the same memory).
#pragma once
#include "common.cuh"

namespace ax {

// ---- 128-bit value in two registers: byte i of the value is byte i of lo (i < 8) or byte i-8 of hi
struct V16 { unsigned long long lo, hi; };

__device__ __forceinline__ V16 shr_bytes(V16 v, uint32_t nb) {          // v >> 8*nb, nb in 0..15
    if (nb >= 8) { v.lo = v.hi >> ((nb - 8) * 8); v.hi = 0; }
    else if (nb) { v.lo = (v.lo >> (nb * 8)) | (v.hi << (64 - nb * 8)); v.hi >>= nb * 8; }
    return v;
}
__device__ __forceinline__ V16 shl_bytes(V16 v, uint32_t nb) {          // v << 8*nb, nb in 1..15
    if (nb >= 8) { v.hi = v.lo << ((nb - 8) * 8); v.lo = 0; }
    else { v.hi = (v.hi << (nb * 8)) | (v.lo >> (64 - nb * 8)); v.lo <<= nb * 8; }
    return v;
}

// The first min(n, 16) bytes at s as a register value; reads whole aligned 8-byte words, so up to 7 bytes before
// s and after the range are loaded and discarded (output buffers are padded to 16 bytes).
__device__ __forceinline__ V16 load16(const uint8_t* s, uint32_t n) {
    const uint32_t sb = (uint32_t)((uintptr_t)s & 7u), need = sb + (n > 16 ? 16 : n);
    const unsigned long long* p = reinterpret_cast<const unsigned long long*>(s - sb);
    const unsigned long long w0 = p[0];
    const unsigned long long w1 = need > 8 ? p[1] : 0ull;
    const unsigned long long w2 = need > 16 ? p[2] : 0ull;
    V16 v;
    if (sb) { const uint32_t sh = sb * 8; v.lo = (w0 >> sh) | (w1 << (64 - sh)); v.hi = (w1 >> sh) | (w2 << (64 - sh)); }
    else { v.lo = w0; v.hi = w1; }
    return v;
}

// Store the first n (<= 16) bytes of v at q with naturally aligned 1/2/4/8-byte stores, nothing outside [q, q+n).
__device__ __forceinline__ void store16(uint8_t* q, V16 v, uint32_t n) {
    if (((uintptr_t)q & 1) && n >= 1) { *q = (uint8_t)v.lo; v = shr_bytes(v, 1); q += 1; n -= 1; }
    if (((uintptr_t)q & 2) && n >= 2) { *reinterpret_cast<uint16_t*>(q) = (uint16_t)v.lo; v = shr_bytes(v, 2); q += 2; n -= 2; }
    if (((uintptr_t)q & 4) && n >= 4) { *reinterpret_cast<uint32_t*>(q) = (uint32_t)v.lo; v = shr_bytes(v, 4); q += 4; n -= 4; }
    if (n >= 8) { *reinterpret_cast<unsigned long long*>(q) = v.lo; v.lo = v.hi; q += 8; n -= 8; }
    if (n >= 8) { *reinterpret_cast<unsigned long long*>(q) = v.lo; return; }
    if (n & 4) { *reinterpret_cast<uint32_t*>(q) = (uint32_t)v.lo; v.lo >>= 32; q += 4; }
    if (n & 2) { *reinterpret_cast<uint16_t*>(q) = (uint16_t)v.lo; v.lo >>= 16; q += 2; }
    if (n & 1) *q = (uint8_t)v.lo;
}

// The same contract as store16 (exactly the bytes [q, q+n), n in 1..16, naturally aligned 1/2/4-byte stores), built for
// latency instead of store count: the value is shifted once to the destination's phase inside its 4-byte word (five
// words, independent funnel shifts) and every possible piece — up to three head bytes, four whole words, up to three
// tail bytes — is a predicated store of one of them, so nothing waits on the previous piece (store16's pieces are a
// chain of shifts).  Used for the shared-memory image of the tile pass, where a warp's stores are its critical path.
__device__ __forceinline__ void place16(uint8_t* q, V16 v, uint32_t n) {
    const uint32_t a = (uint32_t)(uintptr_t)q & 3u, sh = a * 8u, e = a + n;           // e: end byte (exclusive) relative to word 0
    uint8_t* const q0 = q - a;
    const uint32_t s0 = (uint32_t)v.lo, s1 = (uint32_t)(v.lo >> 32), s2 = (uint32_t)v.hi, s3 = (uint32_t)(v.hi >> 32);
    const uint32_t w0 = s0 << sh, w1 = __funnelshift_l(s0, s1, sh), w2 = __funnelshift_l(s1, s2, sh),
                   w3 = __funnelshift_l(s2, s3, sh), w4 = __funnelshift_l(s3, 0u, sh);
    // word 0: bytes [a, min(4, e))
    const uint32_t h = e < 4u ? e : 4u;
    if (a == 0u && h == 4u) *reinterpret_cast<uint32_t*>(q0) = w0;
    else {
        uint32_t p = a;
        if ((p & 1u) && p < h) { q0[p] = (uint8_t)(w0 >> (8u * p)); ++p; }
        if (p + 2u <= h) { *reinterpret_cast<uint16_t*>(q0 + p) = (uint16_t)(w0 >> (8u * p)); p += 2u; }
        if (p < h) q0[p] = (uint8_t)(w0 >> (8u * p));
    }
    // whole words 1 .. 4
    if (e >= 8u) *reinterpret_cast<uint32_t*>(q0 + 4) = w1;
    if (e >= 12u) *reinterpret_cast<uint32_t*>(q0 + 8) = w2;
    if (e >= 16u) *reinterpret_cast<uint32_t*>(q0 + 12) = w3;
    if (e >= 20u) *reinterpret_cast<uint32_t*>(q0 + 16) = w4;     // (n = 16, a = ... never: e <= 19; kept for completeness)
    // tail: bytes [4k, e) of word k = e / 4 >= 1
    const uint32_t k = e >> 2, t = e & 3u;
    if (k >= 1u && t) {
        const uint32_t wk = k == 1u ? w1 : k == 2u ? w2 : k == 3u ? w3 : w4;
        uint8_t* const qk = q0 + 4u * k;
        if (t & 2u) *reinterpret_cast<uint16_t*>(qk) = (uint16_t)wk;
        if (t & 1u) qk[t & 2u] = (uint8_t)(wk >> (8u * (t & 2u)));
    }
}

// OR-merge the first n (1..16) bytes of v into ZEROED memory at q with 8-byte reductions (red.global.or.b64): one L2
// operation per aligned word touched (1 + (n-1)/8 on average) instead of one per naturally aligned piece (~3 for a
// 9-byte match).  Measured on B200: the L2 sustains scattered sub-word writes at a rate set by their COUNT
// (DESIGN.md "Match copy").  Bytes outside [q, q+n) are OR-ed with zero, i.e. left as they are; every byte of the
// output is merged exactly once, so OR equals store.  Global memory only.
__device__ __forceinline__ void merge16(uint8_t* q, V16 v, uint32_t n) {
    if (n < 8) { v.lo &= (1ull << (n * 8)) - 1ull; v.hi = 0; }
    else if (n < 16) v.hi &= n == 8 ? 0ull : (1ull << ((n - 8) * 8)) - 1ull;
    const uint32_t sb = (uint32_t)((uintptr_t)q & 7u), sh = sb * 8;
    unsigned long long* p = reinterpret_cast<unsigned long long*>(q - sb);
    unsigned long long w0 = v.lo, w1 = v.hi, w2 = 0ull;
    if (sh) { w0 = v.lo << sh; w1 = (v.lo >> (64 - sh)) | (v.hi << sh); w2 = v.hi >> (64 - sh); }
    asm volatile("red.global.or.b64 [%0], %1;" ::"l"(p), "l"(w0) : "memory");
    if (sb + n > 8) asm volatile("red.global.or.b64 [%0], %1;" ::"l"(p + 1), "l"(w1) : "memory");
    if (sb + n > 16) asm volatile("red.global.or.b64 [%0], %1;" ::"l"(p + 2), "l"(w2) : "memory");
}

// v holds `period` (1..15) valid bytes: extend it periodically to 16 bytes.
__device__ __forceinline__ V16 extend_period(V16 v, uint32_t period) {
    if (period < 8) { v.lo &= (1ull << (period * 8)) - 1ull; v.hi = 0; }
    else if (period == 8) v.hi = 0;
    else v.hi &= (1ull << ((period - 8) * 8)) - 1ull;
    for (uint32_t d = period; d < 16; d <<= 1) { const V16 s = shl_bytes(v, d); v.lo |= s.lo; v.hi |= s.hi; }
    return v;
}

// v = 16 bytes of a pattern whose period divides c (c <= 16): the 16 bytes starting at phase ph (< period).
// (v >> ph) supplies bytes 0 .. 15-ph; (v << (c-ph)) supplies bytes c-ph .. 15; where both do, they agree.
__device__ __forceinline__ V16 pattern_at(V16 v, uint32_t c, uint32_t ph) {
    V16 r = shr_bytes(v, ph);
    if (c - ph < 16) { const V16 l = shl_bytes(v, c - ph); r.lo |= l.lo; r.hi |= l.hi; }
    return r;
}

// One thread copies one short match (len <= SHORT_MAX = 32) through registers: d[i] = s[i mod dist], dist = d - s
// in the output's coordinates (passed in, because d and s may point into different memories).  Loads only bytes of
// [s, s + min(len, dist)).
__device__ __forceinline__ void thread_copy(uint8_t* d, const uint8_t* s, uint32_t len, uint32_t dist) {
    if (dist >= len) {                                   // no overlap
        store16(d, load16(s, len), len > 16 ? 16 : len);
        if (len > 16) store16(d + 16, load16(s + 16, len - 16), len - 16);
    } else if (dist >= 16) {                             // overlap, 16 <= period < len <= 32: [0,dist) then [dist,len) = s[0 ..)
        store16(d, load16(s, 16), 16);
        if (dist > 16) store16(d + 16, load16(s + 16, dist - 16), dist - 16);
        store16(d + dist, load16(s, len - dist), len - dist);
    } else {                                             // period < 16: replicate it in registers; every chunk of
        const V16 v = extend_period(load16(s, dist), dist);   // c = floor(16/period)*period bytes starts at phase 0
        const uint32_t c = (16u / dist) * dist;
        for (uint32_t done = 0; done < len; done += c) store16(d + done, v, len - done < c ? len - done : c);
    }
}

// One warp copies one long match.  same_mem: d and s address the same memory (so that d - s == dist as pointers and
// a step may read what an earlier step stored); otherwise only [s, s+dist) is ever read.
__device__ __forceinline__ void warp_match(uint8_t* d, const uint8_t* s, uint32_t len, uint32_t dist, bool same_mem, uint32_t lane) {
    if (dist >= len) { warp_copy(d, s, len, lane); return; }
    if (dist >= 16) {
        if (same_mem) {
            // after `done` bytes the range [s, s+dist+done) is valid periodic data, so the copied span doubles every
            // step; __syncwarp orders one step's stores before the next step's loads
            uint32_t done = 0;
            while (done < len) {
                const uint32_t n = len - done < dist + done ? len - done : dist + done;
                warp_copy(d + done, s, n, lane);
                done += n;
                __syncwarp();
            }
        } else {
            for (uint32_t done = 0; done < len; done += dist) warp_copy(d + done, s, len - done < dist ? len - done : dist, lane);
        }
        return;
    }
    // period < 16: the 16 bytes at byte x of the match are the periodic pattern at phase x mod period
    const V16 v = extend_period(load16(s, dist), dist);
    const uint32_t c = (16u / dist) * dist;                          // 9..16, a multiple of the period
    uint32_t n = len;
    uint32_t h = (uint32_t)(-(intptr_t)d) & 15u;
    if (h > n) h = n;
    if (lane == 0 && h) store16(d, v, h);
    d += h; n -= h;
    const uint32_t nvec = n >> 4;
    uint4* d16 = reinterpret_cast<uint4*>(d);
    for (uint32_t w = lane; w < nvec; w += 32) {
        const V16 r = pattern_at(v, c, (h + 16u * w) % dist);
        d16[w] = make_uint4((uint32_t)r.lo, (uint32_t)(r.lo >> 32), (uint32_t)r.hi, (uint32_t)(r.hi >> 32));
    }
    const uint32_t t = n & 15u;
    if (lane == 31 && t) store16(d + 16u * nvec, pattern_at(v, c, (h + 16u * nvec) % dist), t);
}

// ---- one wave-list entry and the register copy of U of them (wave kernel and pass kernel)
struct Ent { uint32_t mdst, off, len; };

__device__ __forceinline__ Ent load_ent(const Params& P, uint32_t i, uint32_t last) {
    Ent e; e.mdst = 0; e.off = 0; e.len = 0;
    if (i < last) { e.mdst = P.wl_dst[i]; e.off = P.wl_off[i]; e.len = P.wl_len[i]; }
    return e;
}

__device__ __forceinline__ bool is_simple(const Ent& e) {   // one 16-byte register copy, no overlap handling needed
    return e.len != 0 && e.len <= 16 && (e.mdst - e.off) >= e.len;
}

__device__ __forceinline__ void long_matches(uint8_t* out, const Ent& e, uint32_t lane) {
    uint32_t longm = __ballot_sync(0xFFFFFFFFu, e.len > SHORT_MAX);
    while (longm) {
        const int sl = __ffs(longm) - 1; longm &= longm - 1;
        const uint32_t d2 = __shfl_sync(0xFFFFFFFFu, e.mdst, sl), o2 = __shfl_sync(0xFFFFFFFFu, e.off, sl),
                       n2 = __shfl_sync(0xFFFFFFFFu, e.len, sl);
        warp_match(out + d2, out + o2, n2, d2 - o2, true, lane);
    }
}

// e[] already loaded: copy them (warp-converged call).  Phase A issues every source load of the U entries in
// straight-line predicated code (no branch between them) so that U round trips to L2 overlap per thread; phase B
// shifts and merges.  "Simple" = at most 16 bytes and no overlap (two aligned 16-byte words hold the source).
template <int U>
__device__ __forceinline__ void copy_ents(uint8_t* out, const Ent (&e)[U], uint32_t lane) {
    uint4 wa[U], wb[U];
    bool simple[U];
#pragma unroll
    for (int k = 0; k < U; ++k) {
        const uint32_t sb = e[k].off & 15u;
        simple[k] = e[k].len != 0 && e[k].len <= 16 && (e[k].mdst - e[k].off) >= e[k].len;
        const uint4* p = reinterpret_cast<const uint4*>(out + (simple[k] ? (e[k].off & ~15u) : 0u));
        wa[k] = p[0];                                              // out has >= 16 bytes: offset 0 is always readable
        wb[k] = make_uint4(0u, 0u, 0u, 0u);
        if (simple[k] && sb + e[k].len > 16) wb[k] = p[1];
    }
#pragma unroll
    for (int k = 0; k < U; ++k) {
        if (simple[k]) {
            const uint32_t sb = e[k].off & 15u, s = (sb & 7u) * 8;
            const unsigned long long a0 = (unsigned long long)wa[k].x | ((unsigned long long)wa[k].y << 32),
                                     a1 = (unsigned long long)wa[k].z | ((unsigned long long)wa[k].w << 32),
                                     b0 = (unsigned long long)wb[k].x | ((unsigned long long)wb[k].y << 32),
                                     b1 = (unsigned long long)wb[k].z | ((unsigned long long)wb[k].w << 32);
            const unsigned long long x0 = sb < 8 ? a0 : a1, x1 = sb < 8 ? a1 : b0, x2 = sb < 8 ? b0 : b1;
            V16 v;
            if (s) { v.lo = (x0 >> s) | (x1 << (64 - s)); v.hi = (x1 >> s) | (x2 << (64 - s)); } else { v.lo = x0; v.hi = x1; }
            merge16(out + e[k].mdst, v, e[k].len);
        } else if (e[k].len != 0 && e[k].len <= SHORT_MAX) thread_copy(out + e[k].mdst, out + e[k].off, e[k].len, e[k].mdst - e[k].off);
    }
#pragma unroll
    for (int k = 0; k < U; ++k) long_matches(out, e[k], lane);
}

}  // namespace ax
