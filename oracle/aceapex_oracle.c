/* oracle/aceapex_oracle.c — ACEAPEX CPU ORACLE.  TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, host-only C.  Shares no code with paper_2606_04268_b200/ (the CUDA path) and is
 * imported only by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs.
 *
 * What it holds (each function cites the passage it follows; byte layout = docs/FORMAT.md):
 *   orc_decode_seq   the DEFINITION of the decoded result: walk cmd[] in sequence, copy literal runs,
 *                    copy matches from their absolute source, ascending          PAPER.md:43 (§3.1), :53 (§3.2)
 *   orc_decode_mt    the paper's block-parallel CPU decoder (baseline only)      PAPER.md:45 (§3.1)
 *   orc_encode       greedy hash-chain encoder: absolute offsets, 1 MB blocks (:49),
 *                    chain flattening (:57-63, §3.3), depth limit (:228, §7.4).  Workload producer:
 *                    its match CHOICES are this repo's (paper silent) => "parity unpinned" for
 *                    ratio / depth profile; its OUTPUT is pinned by invariants I0-I6 and round trip.
 *   orc_validate     invariants I0-I4 over a serialized stream, recomputing depth by the recursive
 *                    definition of PAPER.md:155 (§7.1) (with dep = paper level + 1, Q10)
 *   orc_asap         invariant I5: wave-by-wave ASAP simulation of PAPER.md:194 ("within each level,
 *                    tokens are independent"); the round a match fires in must equal its stored dep
 *
 * Parity pins (tests/test_oracle_*.py): the paper's 5 000/5 100/5 300 example, the
 * A->B->C flattening example, the cross-block limitation, memset /
 * memcpy special cases, a pure-Python byte loop on fuzzed streams, round trip against generator bytes.
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <stdatomic.h>
#include <pthread.h>
#include <sched.h>
#include <sys/mman.h>

enum { ORC_OK = 0, ORC_E_MAGIC = -1, ORC_E_VERSION = -2, ORC_E_TRUNCATED = -3, ORC_E_HEADER = -4,
       ORC_E_CAPACITY = -5, ORC_E_NOMEM = -6, ORC_E_ARG = -7,
       ORC_E_I1 = -11, ORC_E_I2 = -12, ORC_E_I3 = -13, ORC_E_I4 = -14, ORC_E_I5 = -15 };

enum { FLAG_FLATTENED = 1, FLAG_DEPTH_LIMITED = 2, FLAG_HAS_DEP = 4 };
#define HDR_BYTES 64u
#define DIR_BYTES 16u
#define HIST_BYTES 16u
#define MAXLEN 65535u
#define NONE 0xFFFFFFFFu

static inline uint16_t rd16(const uint8_t* p) { uint16_t v; memcpy(&v, p, 2); return v; }
static inline uint32_t rd32(const uint8_t* p) { uint32_t v; memcpy(&v, p, 4); return v; }
static inline uint64_t rd64(const uint8_t* p) { uint64_t v; memcpy(&v, p, 8); return v; }
static inline void wr16(uint8_t* p, uint16_t v) { memcpy(p, &v, 2); }
static inline void wr32(uint8_t* p, uint32_t v) { memcpy(p, &v, 4); }
static inline void wr64(uint8_t* p, uint64_t v) { memcpy(p, &v, 8); }
static inline uint64_t pad16(uint64_t x) { return (x + 15) & ~(uint64_t)15; }
static inline uint64_t pad128(uint64_t x) { return (x + 127) & ~(uint64_t)127; }

/* ------------------------------------------------------------------------------------------------
 * Stream view (I0: header / directory consistency).  docs/FORMAT.md.
 * ---------------------------------------------------------------------------------------------- */
typedef struct {
    const uint8_t* base; uint64_t size;
    uint32_t flags, block_size, n_blocks, min_match, depth_limit, max_depth;
    uint64_t raw_size, total_seq, total_lit;
    const uint8_t* dir; const uint8_t* hist;
} view_t;

typedef struct { const uint8_t *cmd, *len, *dep, *off, *lit; uint32_t n_seq, n_lit; uint64_t out_base, raw_len; } blk_t;

static int view_open(view_t* v, const uint8_t* c, uint64_t size) {
    if (size < HDR_BYTES) return ORC_E_TRUNCATED;
    if (memcmp(c, "ACEAPEX1", 8) != 0) return ORC_E_MAGIC;
    if (rd32(c + 8) != 1) return ORC_E_VERSION;
    v->base = c; v->size = size;
    v->flags = rd32(c + 12); v->raw_size = rd64(c + 16); v->block_size = rd32(c + 24);
    v->n_blocks = rd32(c + 28); v->min_match = rd32(c + 32); v->depth_limit = rd32(c + 36);
    v->max_depth = rd32(c + 40); v->total_seq = rd64(c + 48); v->total_lit = rd64(c + 56);
    if (v->block_size == 0 || v->raw_size > 0xFFFFFFFFull || v->max_depth > 65535) return ORC_E_HEADER;
    uint64_t nb = (v->raw_size + v->block_size - 1) / v->block_size;
    if (nb != v->n_blocks) return ORC_E_HEADER;
    uint64_t meta = HDR_BYTES + (uint64_t)DIR_BYTES * nb + (uint64_t)HIST_BYTES * (v->max_depth + 1ull);
    if (pad128(meta) > size) return ORC_E_TRUNCATED;
    v->dir = c + HDR_BYTES; v->hist = v->dir + (uint64_t)DIR_BYTES * nb;
    uint64_t prev_end = pad128(meta), ts = 0, tl = 0;
    for (uint64_t b = 0; b < nb; ++b) {
        uint64_t po = rd64(v->dir + 16 * b); uint32_t ns = rd32(v->dir + 16 * b + 8), nl = rd32(v->dir + 16 * b + 12);
        if ((po & 127) || po < prev_end) return ORC_E_HEADER;
        uint64_t bytes = 3 * pad16(2ull * ns) + pad16(4ull * ns) + pad16(nl);
        if (po > size || bytes > size - po) return ORC_E_TRUNCATED;
        prev_end = po + bytes; ts += ns; tl += nl;
    }
    if (ts != v->total_seq || tl != v->total_lit) return ORC_E_HEADER;
    return ORC_OK;
}
static void view_block(const view_t* v, uint64_t b, blk_t* k) {
    uint64_t po = rd64(v->dir + 16 * b);
    k->n_seq = rd32(v->dir + 16 * b + 8); k->n_lit = rd32(v->dir + 16 * b + 12);
    const uint8_t* p = v->base + po;
    k->cmd = p; p += pad16(2ull * k->n_seq);
    k->len = p; p += pad16(2ull * k->n_seq);
    k->dep = p; p += pad16(2ull * k->n_seq);
    k->off = p; p += pad16(4ull * k->n_seq);
    k->lit = p;
    k->out_base = b * (uint64_t)v->block_size;
    uint64_t rem = v->raw_size - k->out_base;
    k->raw_len = rem < v->block_size ? rem : v->block_size;
}

uint64_t orc_raw_size(const uint8_t* comp, uint64_t size) {
    view_t v; if (view_open(&v, comp, size)) return (uint64_t)-1; return v.raw_size;
}

/* ------------------------------------------------------------------------------------------------
 * (c1) Sequential decoder — the plain definition.  PAPER.md:53 "processes cmd[] in sequence";
 * PAPER.md:43 "absolute position in the decompressed output".  An overlapping source
 * (off + len > p) reads bytes this same match just wrote: ascending byte copy (Q3).
 * dep[] is ignored.
 * ---------------------------------------------------------------------------------------------- */
static int decode_block(const view_t* v, uint64_t b, uint8_t* out) {
    blk_t k; view_block(v, b, &k);
    uint64_t p = k.out_base, end = k.out_base + k.raw_len, li = 0;
    for (uint32_t j = 0; j < k.n_seq; ++j) {
        uint32_t c = rd16(k.cmd + 2 * j), L = rd16(k.len + 2 * j);
        if (c > end - p || c > k.n_lit - li) return ORC_E_I1;
        for (uint32_t i = 0; i < c; ++i) out[p + i] = k.lit[li + i];
        p += c; li += c;
        if (L) {
            uint64_t o = rd32(k.off + 4 * j);
            if (o >= p) return ORC_E_I2;
            if (L > end - p) return ORC_E_I1;
            for (uint32_t i = 0; i < L; ++i) out[p + i] = out[o + i];
            p += L;
        }
    }
    if (p != end || li != k.n_lit) return ORC_E_I1;
    return ORC_OK;
}

int orc_decode_seq(const uint8_t* comp, uint64_t size, uint8_t* out, uint64_t cap) {
    view_t v; int rc = view_open(&v, comp, size); if (rc) return rc;
    if (cap < v.raw_size) return ORC_E_CAPACITY;
    for (uint64_t b = 0; b < v.n_blocks; ++b) { rc = decode_block(&v, b, out); if (rc) return rc; }
    return ORC_OK;
}

/* ------------------------------------------------------------------------------------------------
 * Thread-parallel decoder (reported baseline).  PAPER.md:45: "threads each process a subset of
 * blocks, with inter-block dependencies handled by processing blocks in order while threads work
 * ahead on their own non-dependent blocks".  Blocks are handed out in increasing order; before a
 * match reads an earlier block b' the thread waits on done[b'] (release/acquire).
 * ---------------------------------------------------------------------------------------------- */
typedef struct { const view_t* v; uint8_t* out; atomic_uint next; atomic_uchar* done; atomic_int err; } mt_t;

static void* mt_worker(void* arg) {
    mt_t* m = (mt_t*)arg; const view_t* v = m->v; uint8_t* out = m->out;
    for (;;) {
        uint32_t b = atomic_fetch_add(&m->next, 1);
        if (b >= v->n_blocks) break;
        blk_t k; view_block(v, b, &k);
        uint64_t p = k.out_base, end = k.out_base + k.raw_len, li = 0; int rc = ORC_OK;
        for (uint32_t j = 0; j < k.n_seq && !rc; ++j) {
            uint32_t c = rd16(k.cmd + 2 * j), L = rd16(k.len + 2 * j);
            if (c > end - p || c > k.n_lit - li) { rc = ORC_E_I1; break; }
            memcpy(out + p, k.lit + li, c); p += c; li += c;
            if (L) {
                uint64_t o = rd32(k.off + 4 * j);
                if (o >= p) { rc = ORC_E_I2; break; }
                if (L > end - p) { rc = ORC_E_I1; break; }
                if (o < k.out_base) {
                    uint64_t last = (o + L <= k.out_base ? o + L : k.out_base) - 1;
                    for (uint64_t bb = o / v->block_size; bb <= last / v->block_size; ++bb)
                        while (!atomic_load_explicit(&m->done[bb], memory_order_acquire)) {
                            if (atomic_load(&m->err)) return NULL;
                            sched_yield();
                        }
                }
                if (o + L <= p) memcpy(out + p, out + o, L);
                else for (uint32_t i = 0; i < L; ++i) out[p + i] = out[o + i];
                p += L;
            }
        }
        if (!rc && (p != end || li != k.n_lit)) rc = ORC_E_I1;
        if (rc) { atomic_store(&m->err, rc); return NULL; }
        atomic_store_explicit(&m->done[b], 1, memory_order_release);
    }
    return NULL;
}

int orc_decode_mt(const uint8_t* comp, uint64_t size, uint8_t* out, uint64_t cap, int threads) {
    view_t v; int rc = view_open(&v, comp, size); if (rc) return rc;
    if (cap < v.raw_size) return ORC_E_CAPACITY;
    if (threads < 1) threads = 1;
    if (threads > 256) threads = 256;
    mt_t m; m.v = &v; m.out = out; atomic_init(&m.next, 0); atomic_init(&m.err, 0);
    m.done = calloc(v.n_blocks + 1, sizeof(atomic_uchar)); if (!m.done) return ORC_E_NOMEM;
    pthread_t th[256];
    for (int t = 0; t < threads; ++t) pthread_create(&th[t], NULL, mt_worker, &m);
    for (int t = 0; t < threads; ++t) pthread_join(th[t], NULL);
    free(m.done);
    return atomic_load(&m.err);
}

/* ------------------------------------------------------------------------------------------------
 * (c2) Encoder.  Paper gives principles only; the algorithm below is DESIGN.md §"Oracle encoder".
 * ---------------------------------------------------------------------------------------------- */
typedef struct {
    uint32_t block_size;     /* B; 1 MB = 2^20                                   */
    uint32_t min_match;      /* MIN = 4 (BASELINE config 0)                                    */
    uint32_t max_chain;      /* candidates walked per position (default 32)                    */
    uint64_t window;         /* max distance p - c; 0 = unlimited ("global view") */
    uint32_t flatten;        /* chain flattening on/off                          */
    uint32_t depth_limit;    /* D; 0 = unlimited                                */
    uint32_t prefer_shallow; /* tie-break knob: among equal lengths take the smaller dep       */
    uint32_t hash_bits;      /* 0 = auto                                                       */
} orc_enc_params;

/* Large zero-filled arrays on transparent huge pages (allocation detail only: random probes into
 * multi-GB tables are TLB-bound on 4 KB pages). */
static void* big_alloc(uint64_t bytes) {
    if (!bytes) bytes = 1;
    void* p = mmap(NULL, bytes, PROT_READ | PROT_WRITE, MAP_PRIVATE | MAP_ANONYMOUS, -1, 0);
    if (p == MAP_FAILED) return NULL;
#ifdef MADV_HUGEPAGE
    madvise(p, bytes, MADV_HUGEPAGE);
#endif
    return p;
}
static void big_free(void* p, uint64_t bytes) { if (p) munmap(p, bytes ? bytes : 1); }

typedef struct { uint8_t* p; uint64_t n, cap; } vec_t;
static int vec_push(vec_t* v, const void* src, uint64_t bytes) {
    if (v->n + bytes > v->cap) {
        uint64_t nc = v->cap ? v->cap : 4096; while (nc < v->n + bytes) nc += nc / 2 + 4096;
        uint8_t* q = realloc(v->p, nc); if (!q) return -1; v->p = q; v->cap = nc;
    }
    memcpy(v->p + v->n, src, bytes); v->n += bytes; return 0;
}

static inline uint32_t hash4(const uint8_t* p, uint32_t hb) { return (rd32(p) * 2654435761u) >> (32 - hb); }

int orc_encode(const uint8_t* in, uint64_t n, const orc_enc_params* P, uint8_t** out, uint64_t* out_size) {
    if (!P || !out || !out_size || P->block_size == 0 || n > 0xFFFFFFFFull || P->min_match < 1) return ORC_E_ARG;
    const uint32_t B = P->block_size, MIN = P->min_match, D = P->depth_limit ? P->depth_limit : 65535u;
    if (D > 65535u) return ORC_E_ARG;
    const uint64_t WIN = P->window ? P->window : ~0ull;
    uint32_t hb = P->hash_bits; if (!hb) { hb = 12; while (hb < 24 && (1ull << hb) < n) ++hb; }
    const uint64_t nb = (n + B - 1) / B;
    /* Hash chains, most recent first, truncated at max_chain entries: stored as one row of K = max_chain
     * positions per hash value (row[0] = most recent).  Same candidate set and order as walking a linked
     * chain for max_chain steps; the row form costs one cache miss per lookup instead of one per step.
     * Each row is a ring: cur[h] is the slot of the most recent entry, older entries follow backwards. */
    const uint32_t K = P->max_chain ? (P->max_chain > 64 ? 64 : P->max_chain) : 1;
    uint32_t cand[64];
    const uint64_t head_bytes = (sizeof(uint32_t) * (uint64_t)K) << hb, bd_bytes = 2 * (n + 1);
    uint32_t* head = big_alloc(head_bytes);
    uint8_t* cur = big_alloc(1ull << hb);
    uint16_t* bd   = big_alloc(bd_bytes);                    /* byte depth: 0 literal, d = written by a depth-d match */
    uint32_t* root = malloc(sizeof(uint32_t) * (uint64_t)B);  /* current block only: resolved source of a match byte   */
    uint32_t* bseq = calloc(nb + 1, 4); uint32_t* blit = calloc(nb + 1, 4);
    uint64_t* hcnt = calloc(65536, 8); uint64_t* hbytes = calloc(65536, 8);
    vec_t vc = {0}, vl = {0}, vd = {0}, vo = {0}, vlit = {0};
    int rc = ORC_E_NOMEM;
    if (!head || !cur || !bd || !root || !bseq || !blit || !hcnt || !hbytes) goto done;
    memset(head, 0xFF, head_bytes);

#define EMIT(cv, lv, ov, dv) do { uint16_t c_ = (uint16_t)(cv), l_ = (uint16_t)(lv), d_ = (uint16_t)(dv); uint32_t o_ = (uint32_t)(ov); \
        if (vec_push(&vc, &c_, 2) || vec_push(&vl, &l_, 2) || vec_push(&vd, &d_, 2) || vec_push(&vo, &o_, 4)) goto done; \
        bseq[b]++; if (c_) { hcnt[0]++; hbytes[0] += c_; } if (l_) { hcnt[d_]++; hbytes[d_] += l_; } } while (0)
#define INSERT(x) do { if ((uint64_t)(x) + 4 <= n) { uint32_t h_ = hash4(in + (x), hb); \
        uint8_t k_ = (uint8_t)((cur[h_] + 1u) % K); cur[h_] = k_; head[(uint64_t)h_ * K + k_] = (uint32_t)(x); } } while (0)

    for (uint64_t b = 0; b < nb; ++b) {
        const uint64_t base = b * B, end = base + B < n ? base + B : n;
        uint64_t p = base, run_start = base;
        while (p < end) {
            uint32_t bestL = 0, bestOff = 0, bestDep = 0;
            if (p + MIN <= end && p + 4 <= n) {
                const uint32_t hp = hash4(in + p, hb), c0 = cur[hp];
                const uint32_t* row = head + (uint64_t)hp * K;
                const uint32_t p4 = rd32(in + p);
                uint32_t ncand = 0;
                for (; ncand < K && ncand < 64; ++ncand) {                 /* resolve sources, start their cache misses */
                    const uint32_t c = row[(c0 + K - ncand) % K];
                    if (c == NONE || p - c > WIN) break;                  /* chain is most-recent-first */
                    uint64_t s = c;
                    if (P->flatten && c >= base && bd[c] != 0) s = root[c - base];   /* step to the resolved source */
                    cand[ncand] = (uint32_t)s;
                    __builtin_prefetch(in + s); __builtin_prefetch(bd + s);
                }
                for (uint32_t steps = 0; steps < ncand; ++steps) {
                    const uint64_t s = cand[steps];
                    /* pruning only: L >= MIN >= 4 needs the first four bytes equal; a candidate that
                     * mismatches at index bestL cannot be strictly longer */
                    if (MIN >= 4 && rd32(in + s) != p4) continue;
                    if (bestL && !P->prefer_shallow && p + bestL < end && in[s + bestL] != in[p + bestL]) continue;
                    uint32_t L = 0, dmax = 0;
                    while (p + L < end && L < MAXLEN) {
                        uint64_t q = s + L;
                        if (q < p) {                                       /* a byte that exists before this match */
                            if (P->flatten && q >= base && bd[q] != 0) break;   /* would read a same-block match byte */
                            if ((uint32_t)bd[q] + 1 > D) break;            /* would exceed the depth limit */
                            if (in[q] != in[p + L]) break;
                            if (bd[q] > dmax) dmax = bd[q];
                        } else {                                           /* self-overlap: this match's own output */
                            if (in[q] != in[p + L]) break;
                        }
                        ++L;
                    }
                    if (L >= MIN && (L > bestL || (P->prefer_shallow && L == bestL && 1 + dmax < bestDep))) {
                        bestL = L; bestOff = (uint32_t)s; bestDep = 1 + dmax;
                    }
                }
            }
            if (bestL) {
                uint64_t run = p - run_start;
                while (run > MAXLEN) { if (vec_push(&vlit, in + run_start, MAXLEN)) goto done; EMIT(MAXLEN, 0, 0, 0); blit[b] += MAXLEN; run_start += MAXLEN; run -= MAXLEN; }
                if (vec_push(&vlit, in + run_start, run)) goto done;
                blit[b] += (uint32_t)run;
                EMIT(run, bestL, bestOff, bestDep);
                const uint64_t period = p - bestOff;
                for (uint32_t i = 0; i < bestL; ++i) {
                    bd[p + i] = (uint16_t)bestDep;
                    root[p + i - base] = (bestOff + (uint64_t)i >= p) ? (uint32_t)(bestOff + i % period) : bestOff + i;
                    INSERT(p + i);
                }
                p += bestL; run_start = p;
            } else {
                bd[p] = 0; INSERT(p); ++p;
            }
        }
        {   /* trailing literals; every block ends up with at least one sequence */
            uint64_t run = end - run_start;
            while (run > MAXLEN) { if (vec_push(&vlit, in + run_start, MAXLEN)) goto done; EMIT(MAXLEN, 0, 0, 0); blit[b] += MAXLEN; run_start += MAXLEN; run -= MAXLEN; }
            if (run || bseq[b] == 0) { if (vec_push(&vlit, in + run_start, run)) goto done; blit[b] += (uint32_t)run; EMIT(run, 0, 0, 0); }
        }
    }
    {   /* serialize (docs/FORMAT.md) */
        uint32_t max_depth = 0; for (uint32_t d = 1; d < 65536; ++d) if (hcnt[d]) max_depth = d;
        uint64_t total_seq = vc.n / 2, total_lit = vlit.n;
        uint64_t meta = pad128(HDR_BYTES + DIR_BYTES * nb + (uint64_t)HIST_BYTES * (max_depth + 1ull));
        uint64_t tot = meta;
        for (uint64_t b = 0; b < nb; ++b) tot += pad128(3 * pad16(2ull * bseq[b]) + pad16(4ull * bseq[b]) + pad16(blit[b]));
        uint8_t* o = calloc(tot ? tot : 1, 1); if (!o) goto done;
        memcpy(o, "ACEAPEX1", 8); wr32(o + 8, 1);
        wr32(o + 12, (P->flatten ? FLAG_FLATTENED : 0) | (P->depth_limit ? FLAG_DEPTH_LIMITED : 0) | FLAG_HAS_DEP);
        wr64(o + 16, n); wr32(o + 24, B); wr32(o + 28, (uint32_t)nb); wr32(o + 32, MIN); wr32(o + 36, P->depth_limit);
        wr32(o + 40, max_depth); wr32(o + 44, 0); wr64(o + 48, total_seq); wr64(o + 56, total_lit);
        uint8_t* hist = o + HDR_BYTES + DIR_BYTES * nb;
        for (uint32_t d = 0; d <= max_depth; ++d) { wr32(hist + 16 * d, (uint32_t)hcnt[d]); wr64(hist + 16 * d + 8, hbytes[d]); }
        uint64_t po = meta, sj = 0, lj = 0;
        for (uint64_t b = 0; b < nb; ++b) {
            uint32_t ns = bseq[b], nl = blit[b];
            wr64(o + HDR_BYTES + 16 * b, po); wr32(o + HDR_BYTES + 16 * b + 8, ns); wr32(o + HDR_BYTES + 16 * b + 12, nl);
            uint8_t* q = o + po;
            memcpy(q, vc.p + 2 * sj, 2ull * ns); q += pad16(2ull * ns);
            memcpy(q, vl.p + 2 * sj, 2ull * ns); q += pad16(2ull * ns);
            memcpy(q, vd.p + 2 * sj, 2ull * ns); q += pad16(2ull * ns);
            memcpy(q, vo.p + 4 * sj, 4ull * ns); q += pad16(4ull * ns);
            memcpy(q, vlit.p + lj, nl);
            sj += ns; lj += nl;
            po += pad128(3 * pad16(2ull * ns) + pad16(4ull * ns) + pad16(nl));
        }
        *out = o; *out_size = tot; rc = ORC_OK;
    }
done:
    big_free(head, head_bytes); big_free(cur, 1ull << hb); big_free(bd, bd_bytes); free(root); free(bseq); free(blit); free(hcnt); free(hbytes);
    free(vc.p); free(vl.p); free(vd.p); free(vo.p); free(vlit.p);
    return rc;
}
void orc_free(void* p) { free(p); }

/* ------------------------------------------------------------------------------------------------
 * (c3) Validator: I0 (view_open), I1-I4, independent of the encoder's state.
 *   I1  per block: sum(cmd+len) = raw_len, sum(cmd) = n_lit
 *   I2  per match: len in [min_match, 65535]; off < mdst; placeholder has off = dep = 0
 *   I3  FLATTENED: every effective source byte inside the own block is a literal
 *   I4  stored dep = 1 + max byte depth over the effective source range [off, min(off+len, mdst))
 *       (PAPER.md:155 with dep = level + 1); DEPTH_LIMITED => dep <= D;
 *       header max_depth and depth histogram agree with the recount.
 * ---------------------------------------------------------------------------------------------- */
typedef struct {
    uint64_t raw_bytes, comp_bytes, lit_bytes, match_bytes, match_src_bytes, n_seq, n_match;
    uint32_t n_blocks, block_size, max_depth, depth_limit, flags, fail_block; uint64_t fail_seq;
} orc_report;

int orc_validate(const uint8_t* comp, uint64_t size, orc_report* R) {
    view_t v; int rc = view_open(&v, comp, size); if (rc) return rc;
    orc_report r; memset(&r, 0, sizeof r);
    r.raw_bytes = v.raw_size; r.comp_bytes = size; r.n_blocks = v.n_blocks; r.block_size = v.block_size;
    r.depth_limit = v.depth_limit; r.flags = v.flags;
    uint16_t* bd = calloc(v.raw_size + 1, 2);
    uint64_t* hc = calloc(65536, 8); uint64_t* hbv = calloc(65536, 8);
    if (!bd || !hc || !hbv) { free(bd); free(hc); free(hbv); return ORC_E_NOMEM; }
    for (uint64_t b = 0; b < v.n_blocks && !rc; ++b) {
        blk_t k; view_block(&v, b, &k);
        uint64_t p = k.out_base, end = p + k.raw_len, li = 0;
        for (uint32_t j = 0; j < k.n_seq; ++j) {
            uint32_t c = rd16(k.cmd + 2 * j), L = rd16(k.len + 2 * j), dp = rd16(k.dep + 2 * j);
            uint64_t o = rd32(k.off + 4 * j);
            r.fail_block = (uint32_t)b; r.fail_seq = j;
            if (c > end - p || c > k.n_lit - li) { rc = ORC_E_I1; break; }
            p += c; li += c;                                   /* literal bytes: bd stays 0 */
            if (c) { hc[0]++; hbv[0] += c; }
            if (L == 0) { if (o != 0 || dp != 0) { rc = ORC_E_I2; break; } continue; }
            if (L < v.min_match || o >= p) { rc = ORC_E_I2; break; }
            if (L > end - p) { rc = ORC_E_I1; break; }
            uint64_t se = o + L < p ? o + L : p; uint32_t dmax = 0;
            for (uint64_t q = o; q < se; ++q) {
                if ((v.flags & FLAG_FLATTENED) && q >= k.out_base && bd[q] != 0) { rc = ORC_E_I3; break; }
                if (bd[q] > dmax) dmax = bd[q];
            }
            if (rc) break;
            if (dp != dmax + 1 || dp > v.max_depth) { rc = ORC_E_I4; break; }
            if ((v.flags & FLAG_DEPTH_LIMITED) && dp > v.depth_limit) { rc = ORC_E_I4; break; }
            for (uint32_t i = 0; i < L; ++i) bd[p + i] = (uint16_t)dp;
            hc[dp]++; hbv[dp] += L; r.n_match++; r.match_bytes += L; r.match_src_bytes += se - o;
            if (dp > r.max_depth) r.max_depth = dp;
            p += L;
        }
        if (!rc && (p != end || li != k.n_lit)) rc = ORC_E_I1;
        r.n_seq += k.n_seq; r.lit_bytes += k.n_lit;
    }
    if (!rc) {
        if (r.max_depth != v.max_depth) rc = ORC_E_I4;
        for (uint32_t d = 0; d <= v.max_depth && !rc; ++d)
            if (rd32(v.hist + 16 * d) != (uint32_t)hc[d] || rd64(v.hist + 16 * d + 8) != hbv[d]) rc = ORC_E_I4;
        if (!rc) { r.fail_block = 0; r.fail_seq = 0; }
    }
    free(bd); free(hc); free(hbv);
    if (R) *R = r;
    return rc;
}

/* ------------------------------------------------------------------------------------------------
 * I5: ASAP wave simulation (small inputs; O(rounds * n_seq)).  Round 0 places every literal
 * (Q11).  In round r >= 1 every unfired match whose effective source bytes were all
 * written in rounds < r fires.  PAPER.md:155 (levels), :194 (independence within a level).
 * Returns the number of rounds (= max_depth) or a negative error; out receives the wave-built bytes.
 * ---------------------------------------------------------------------------------------------- */
int64_t orc_asap(const uint8_t* comp, uint64_t size, uint8_t* out, uint64_t cap) {
    view_t v; int rc = view_open(&v, comp, size); if (rc) return rc;
    if (cap < v.raw_size) return ORC_E_CAPACITY;
    uint64_t ns = v.total_seq;
    uint32_t* wr = malloc(4 * (v.raw_size + 1));                 /* round a byte was written in; NONE = not yet */
    uint64_t* mdst = malloc(8 * (ns + 1)); uint32_t* mo = malloc(4 * (ns + 1)); uint16_t* ml = malloc(2 * (ns + 1));
    uint16_t* md = malloc(2 * (ns + 1)); uint8_t* fired = calloc(ns + 1, 1);
    if (!wr || !mdst || !mo || !ml || !md || !fired) { rc = ORC_E_NOMEM; goto out_; }
    memset(wr, 0xFF, 4 * (v.raw_size + 1));
    uint64_t t = 0, left = 0;
    for (uint64_t b = 0; b < v.n_blocks; ++b) {
        blk_t k; view_block(&v, b, &k);
        uint64_t p = k.out_base, end = p + k.raw_len, li = 0;
        for (uint32_t j = 0; j < k.n_seq; ++j, ++t) {
            uint32_t c = rd16(k.cmd + 2 * j), L = rd16(k.len + 2 * j);
            if (c > end - p || c > k.n_lit - li || L > end - p - c) { rc = ORC_E_I1; goto out_; }
            for (uint32_t i = 0; i < c; ++i) { out[p + i] = k.lit[li + i]; wr[p + i] = 0; }
            p += c; li += c;
            mdst[t] = p; mo[t] = rd32(k.off + 4 * j); ml[t] = (uint16_t)L; md[t] = rd16(k.dep + 2 * j);
            if (L) { if (mo[t] >= p) { rc = ORC_E_I2; goto out_; } ++left; } else fired[t] = 1;
            p += L;
        }
        if (p != end) { rc = ORC_E_I1; goto out_; }
    }
    uint32_t r = 0;
    while (left) {
        ++r; uint64_t nf = 0;
        for (uint64_t i = 0; i < ns; ++i) {
            if (fired[i]) continue;
            uint64_t se = (uint64_t)mo[i] + ml[i] < mdst[i] ? (uint64_t)mo[i] + ml[i] : mdst[i]; int ok = 1;
            for (uint64_t q = mo[i]; q < se; ++q) if (wr[q] >= r) { ok = 0; break; }   /* NONE >= r too */
            if (!ok) continue;
            if (md[i] != r) { rc = ORC_E_I5; goto out_; }
            for (uint32_t x = 0; x < ml[i]; ++x) out[mdst[i] + x] = out[mo[i] + x];
            for (uint32_t x = 0; x < ml[i]; ++x) wr[mdst[i] + x] = r;
            fired[i] = 1; ++nf;
        }
        if (!nf) { rc = ORC_E_I5; goto out_; }
        left -= nf;
    }
    rc = 0;
    free(wr); free(mdst); free(mo); free(ml); free(md); free(fired);
    return (int64_t)r;
out_:
    free(wr); free(mdst); free(mo); free(ml); free(md); free(fired);
    return rc;
}
