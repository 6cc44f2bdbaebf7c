/* include/aceapex.h — C ABI of libaceapex: B200 (sm_100a) GPU decode of the ACEAPEX LZ77 token stream.
 *
 * What is decoded.  ACEAPEX (arxiv 2606.04268) stores back-references as ABSOLUTE positions in the
 * decompressed output (§3.1), cuts the data into 1 MB blocks of four pre-decoded streams
 * lit[] / len[] / off[] / cmd[] (§3.2) and flattens dependency chains at encode time so
 * every match sits at a known dependency depth (PAPER.md:57-63 §3.3, :155 §7.1).  The decoded result is,
 * by definition, what the sequential walk of PAPER.md:53 produces: per block, per sequence, copy the
 * literal run, then copy len bytes from out[off..] in ascending order.  This library reaches exactly
 * that result as: block/token index -> exclusive length scan -> literal scatter -> match copy in an order
 * that respects the dependencies: one wave per dependency depth from bucketed lists or by one streaming
 * pass per depth (§4.4/§7.1), or — for flattened streams — one pass in block order
 * (after chain flattening a match depends on earlier blocks only).  Byte layout of the
 * compressed buffer: docs/FORMAT.md (version 1).
 *
 * Conventions.  No C++ or PyTorch types.  "host" / "device" is stated per pointer.  All functions
 * return 0 (ACEAPEX_OK) or a negative ACEAPEX_E_* code; nothing throws, nothing allocates device memory
 * inside aceapex_decode.  One GPU, no collectives, no CPU fallback: if no CUDA device is usable every
 * entry point that needs one returns ACEAPEX_E_CUDA.
 */
#ifndef ACEAPEX_H
#define ACEAPEX_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct aceapex_plan_s aceapex_plan_t; /* opaque; created by aceapex_plan, released by aceapex_free */

enum {
    ACEAPEX_OK = 0,
    ACEAPEX_E_MAGIC = -1,     /* first 8 bytes are not "ACEAPEX1"                                     */
    ACEAPEX_E_VERSION = -2,   /* version field != 1                                                   */
    ACEAPEX_E_TRUNCATED = -3, /* header, directory, histogram or a payload runs past comp_bytes       */
    ACEAPEX_E_HEADER = -4,    /* inconsistent header / directory (sizes, counts, offsets, alignment)  */
    ACEAPEX_E_CAPACITY = -5,  /* out_capacity or scratch_bytes too small                              */
    ACEAPEX_E_ALIGN = -6,     /* a device pointer is not 16-byte aligned                              */
    ACEAPEX_E_CUDA = -7,      /* a CUDA runtime call failed (see aceapex_last_cuda_error)             */
    ACEAPEX_E_ARG = -8,       /* NULL / out-of-range argument                                         */
    ACEAPEX_E_STREAM = -9,    /* token-level fault found on the device (see aceapex_stats.fault_*)    */
    ACEAPEX_E_NOMEM = -10,    /* host allocation failed                                               */
    ACEAPEX_E_NOALLOC_LIMIT = -11 /* aceapex_decode_noalloc: the stream needs more scratch than the static buffer holds */
};

/* phases bitmask of aceapex_decode */
enum {
    ACEAPEX_PHASE_PRE = 1,   /* index + scan + literal scatter + depth bucketing (steps a1-a5)        */
    ACEAPEX_PHASE_MATCH = 2, /* the match-copy waves, depth 1 .. max_depth (steps a6-a7)              */
    ACEAPEX_PHASE_ALL = 3
};

/* wave sequencing strategies (step a7); AUTO picks from the plan's per-depth histogram */
enum {
    ACEAPEX_WAVES_AUTO = 0,
    ACEAPEX_WAVES_LAUNCH = 1,     /* wave lists; one kernel launch per depth on the caller's stream          */
    ACEAPEX_WAVES_GRAPH = 2,      /* the same launches replayed from a cached CUDA graph       */
    ACEAPEX_WAVES_PERSISTENT = 3, /* wave lists; one cooperative kernel, grid barrier between depths         */
    ACEAPEX_WAVES_PASSES = 4,     /* shallow streams (max_depth <= 16, e.g. the depth-limited encoder of PAPER.md:228): no wave
                                     lists; the token stream is re-parsed once per depth, pass p copying the matches with
                                     dep == p (k_pass).  E_ARG from aceapex_set_strategy if max_depth > 16          */
    ACEAPEX_WAVES_CHAIN = 5       /* FLATTENED streams only (after chain flattening no match reads a byte
                                     another match of its own block produced): no wave lists; ONE pass over the token
                                     stream in block order copies every match, a tile waiting until all earlier blocks
                                     are written (k_chain).  E_ARG from aceapex_set_strategy if the header's
                                     FLATTENED flag is clear                                                    */
};

/* device-side token fault bits (aceapex_stats.fault_flags) */
enum {
    ACEAPEX_F_BLOCK_SUM = 1, /* sum(cmd+len) != raw_len[b] or sum(cmd) != n_lit[b]  (I1)               */
    ACEAPEX_F_SOURCE = 2,    /* off >= mdst, or len < min_match                     (I2)               */
    ACEAPEX_F_DEPTH = 4,     /* dep == 0 on a match, dep > max_depth, or counts != depth histogram     */
    ACEAPEX_F_PLACEHOLDER = 8,/* len == 0 with off != 0 or dep != 0                                    */
    ACEAPEX_F_INDEX = 16     /* directory / histogram in comp_dev disagree with what aceapex_plan validated
                                on the host copy (a different or modified buffer): nothing was decoded   */
};

typedef struct {
    uint64_t raw_bytes;       /* N: decompressed size (header)                                         */
    uint64_t comp_bytes;      /* C: size of the compressed buffer                                      */
    uint64_t lit_bytes;       /* Lit: literal bytes (header total_lit)                                 */
    uint64_t match_bytes;     /* M = N - Lit                                                           */
    uint64_t match_src_bytes; /* M_src = sum over matches of min(len, mdst-off); counted on the device
                                 during the decode, 0 before the first one                                 */
    uint64_t n_seq;           /* sequences (header total_seq)                                          */
    uint64_t n_match;         /* matches = sum of depth histogram counts for d >= 1                    */
    uint32_t n_blocks, block_size, min_match, max_depth, depth_limit, flags;
    uint32_t strategy;        /* ACEAPEX_WAVES_* actually used by the last decode (or that AUTO picks) */
    uint32_t n_launches;      /* kernels launched by the last aceapex_decode call                      */
    uint32_t fault_flags;     /* ACEAPEX_F_* bits, read back from the device                           */
    uint32_t fault_block;     /* lowest block index that raised a fault (valid if fault_flags != 0)    */
} aceapex_stats;

/* aceapex_plan — parse and validate header, block directory and depth histogram (docs/FORMAT.md;
 * PAPER.md:49-53), size the scratch, choose the wave strategy.
 *   comp_host  HOST pointer to the whole compressed buffer, comp_bytes long.  Only header, directory and
 *              histogram are read (O(n_blocks + max_depth) bytes); the pointer is not retained.
 *   device     CUDA device ordinal the plan is bound to (queried for SM count / co-residency).
 *   out        receives the plan.  Owned by the library; release with aceapex_free.
 * Errors: E_ARG, E_MAGIC, E_VERSION, E_TRUNCATED, E_HEADER, E_NOMEM, E_CUDA.  *out is NULL on error. */
int aceapex_plan(const void* comp_host, size_t comp_bytes, int device, aceapex_plan_t** out);

/* Bytes the caller must provide.  aceapex_out_bytes = raw size rounded up to 16: kernels load whole aligned
 * 16-byte words of the output and OR-merge aligned 8-byte words of it (red.or with zeros outside the token), so
 * the padding may be read and rewritten with its own value; no byte outside [0, raw_bytes) ever CHANGES, and
 * nothing beyond aceapex_out_bytes is touched. */
size_t aceapex_raw_bytes(const aceapex_plan_t* p);
size_t aceapex_out_bytes(const aceapex_plan_t* p);
size_t aceapex_scratch_bytes(const aceapex_plan_t* p);

/* Force a wave strategy (ACEAPEX_WAVES_*); AUTO restores the plan's own choice.  E_ARG if unknown. */
int aceapex_set_strategy(aceapex_plan_t* p, int strategy);

/* aceapex_decode — enqueue the decode on `stream` and return without synchronising the host.
 *   comp_dev      DEVICE pointer, the same comp_bytes given to aceapex_plan, 16-byte aligned, read only.
 *   out_dev       DEVICE pointer, >= aceapex_out_bytes(p) bytes, 16-byte aligned.  Under every strategy but CHAIN,
 *                 PHASE_PRE first zeroes bytes [0, raw) (short matches are OR-merged into zeros); then bytes
 *                 [0, raw) are written.  Contents on entry do not matter.
 *   scratch_dev   DEVICE pointer, >= aceapex_scratch_bytes(p) bytes, 16-byte aligned.  Contents are
 *                 undefined on entry for PHASE_PRE; PHASE_MATCH alone reuses what PRE left there.
 *   phases        ACEAPEX_PHASE_* mask.  MATCH alone requires a completed PRE on the same scratch and out
 *                 (this is how the match phase is timed alone, the paper's scope: PAPER.md:99, :121).
 *   stream        a cudaStream_t passed as void* (NULL = legacy default stream).
 * All three buffers are owned by the caller and must stay alive until the stream reaches the end of the
 * decode.  One plan must not be in flight on two streams at once.
 * Token-level faults never cause an out-of-bounds access; they are recorded in scratch and surface from
 * aceapex_get_stats as E_STREAM.  Errors here: E_ARG, E_CAPACITY, E_ALIGN, E_CUDA.
 * What is NOT checked: dep[] is trusted for scheduling (the device checks only its range and that the per-depth counts
 * match the header's histogram; under CHAIN also that an in-block source has dep == 1).  A stream whose dep[] understates
 * a match's true depth — with a histogram to match — lets that match read bytes its wave has not written yet: the output
 * is then wrong although every access stays in bounds and no fault is raised.  Recomputing depths is the validator's job
 * (oracle/: invariant I4); a producer that cannot be trusted should be validated before its streams are decoded. */
int aceapex_decode(aceapex_plan_t* p, const void* comp_dev, void* out_dev, size_t out_capacity,
                   void* scratch_dev, size_t scratch_bytes, unsigned phases, void* stream);

/* aceapex_decode_host — the same decode from HOST buffers (end-to-end entry: PAPER.md:121 names the
 * PCIe transfer as the term its timing excludes).  Enqueues on `stream`: H2D copy comp_host -> comp_dev,
 * the full decode, D2H copy out_dev -> out_host (raw_bytes bytes).  comp_host / out_host should be pinned
 * for the copies to be asynchronous; the caller synchronises the stream before reading out_host.
 * comp_dev / out_dev / scratch_dev are caller-owned DEVICE staging buffers, sized and aligned as above.
 * comp_host must hold the bytes the plan was made from (comp_bytes must equal the planned size; a directory or histogram
 * that differs from the planned one is caught on the device and reported as ACEAPEX_F_INDEX, nothing being decoded). */
int aceapex_decode_host(aceapex_plan_t* p, const void* comp_host, size_t comp_bytes, void* out_host,
                        size_t out_host_capacity, void* comp_dev, void* out_dev, size_t out_capacity,
                        void* scratch_dev, size_t scratch_bytes, void* stream);

/* aceapex_get_stats — synchronises `stream` of the last decode, reads the device status words of
 * `scratch_dev` back and fills *s.  Returns E_STREAM if the device recorded a token fault. */
int aceapex_get_stats(aceapex_plan_t* p, const void* scratch_dev, aceapex_stats* s);

/* Depth histogram from the header (PAPER.md:155 levels, dep = level + 1): entry d (0 <= d < cap) gets the
 * number of matches / match bytes at depth d (d = 0: literal runs / literal bytes).  Returns the number
 * of entries available (max_depth + 1) or a negative error. */
int64_t aceapex_depth_hist(const aceapex_plan_t* p, uint64_t* n_match, uint64_t* n_bytes, uint32_t cap);

/* aceapex_decode_noalloc — the full decode (PHASE_ALL) for callers that cannot provide device scratch and must not
 * trigger an allocation (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).  Same
 * kernels, same comp_dev / out_dev / stream meaning as aceapex_decode; the scratch is ONE static device array owned by
 * the library: aceapex_noalloc_max_scratch_bytes() = 16 MiB, held by every GPU that loads the library until the process
 * exits.  A plan whose aceapex_scratch_bytes exceeds that is rejected with ACEAPEX_E_NOALLOC_LIMIT (nothing is launched).
 * The call performs no cudaMalloc / cudaFree / allocating library routine (strategy GRAPH is run as LAUNCH).  Every call
 * on a device shares the array and finds the last call's contents in it; nothing relies on them (the pre-phase resets what
 * must start at zero).  Calls that overlap on the GPU — two streams, two plans, two threads — RACE on the array: one decode
 * at a time per device, and aceapex_get_stats_noalloc (same meaning as aceapex_get_stats) before the next one.
 * Errors: E_ARG (also: current device is not the plan's), E_NOALLOC_LIMIT, E_CAPACITY, E_ALIGN, E_CUDA. */
int aceapex_decode_noalloc(aceapex_plan_t* p, const void* comp_dev, void* out_dev, size_t out_capacity, void* stream);
int aceapex_get_stats_noalloc(aceapex_plan_t* p, aceapex_stats* s);
size_t aceapex_noalloc_max_scratch_bytes(void);

const char* aceapex_strerror(int code);
int aceapex_last_cuda_error(const aceapex_plan_t* p); /* cudaError_t of the last failing CUDA call, else 0 */

void aceapex_free(aceapex_plan_t* p); /* NULL is a no-op; destroys cached graphs; frees no caller buffer */

#ifdef __cplusplus
}
#endif
#endif /* ACEAPEX_H */
