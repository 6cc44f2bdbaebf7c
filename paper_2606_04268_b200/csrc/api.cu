// api.cu — the C ABI of libaceapex (include/aceapex.h): plan (host-side header/directory validation, scratch
// layout, wave strategy), decode (kernel sequencing on the caller's stream), stats.
#include "../../include/aceapex.h"
#include "common.cuh"

#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

namespace ax {
void launch_index(const Params& P, cudaStream_t st);
void launch_tilesum(const Params& P, int grid, cudaStream_t st);
void launch_pre(const Params& P, int grid, cudaStream_t st);
void launch_check_cursors(const Params& P, cudaStream_t st);
cudaError_t pass_configure();
int pass_max_ctas_per_sm();
void launch_pass(const Params& P, uint32_t p, int grid, cudaStream_t st);
void launch_pass_reset(const Params& P, cudaStream_t st);
void launch_litcopy(const Params& P, int grid, cudaStream_t st);
cudaError_t pre_configure();
int pre_max_ctas_per_sm(uint32_t max_depth);
int match_max_ctas_per_sm();
cudaError_t waves_configure();
cudaError_t launch_wave(const Params& P, uint32_t depth, uint32_t n_entries, int max_grid, cudaStream_t st);
cudaError_t launch_waves_persistent(const Params& P, uint32_t d_first, uint32_t d_last, int grid, cudaStream_t st);
cudaError_t chain_configure();
int chain_max_ctas_per_sm();
cudaError_t launch_chain(const Params& P, int grid, cudaStream_t st);
size_t chain_sync_words(uint32_t n_blocks);
}  // namespace ax

using namespace ax;

struct GraphSlot {
    const void* comp; void* out; void* scratch; unsigned phases; int strategy;
    cudaGraphExec_t exec; uint32_t n_launches;
};

struct aceapex_plan_s {
    // header (docs/FORMAT.md)
    uint32_t flags, block_size, n_blocks, min_match, depth_limit, max_depth;
    uint64_t raw_size, total_seq, total_lit, comp_bytes, n_match;
    std::vector<uint64_t> hist_cnt, hist_bytes;     // [max_depth + 1]
    uint32_t lit_q_cap;                             // capacity of the long-literal queue
    uint32_t list_mask;                             // strategy PASSES: sparse depths (listed by the literal pass)
    uint32_t n_tiles_list, n_tiles_stream;          // tiles at TILE_LIST / TILE_STREAM sequences per tile
    // device facts
    int device, n_sm, pre_grid, match_ctas_per_sm, chain_grid, pass_grid;
    // scratch layout (byte offsets)
    size_t o_status, o_wave_off, o_cursor, o_blocks, o_tiles, o_tblk, o_chain, o_litq, o_dst, o_off, o_len, scratch_bytes;
    int strategy_auto, strategy_forced;
    uint32_t last_launches; int last_strategy; bool last_had_match;
    int last_cuda;
    cudaStream_t last_stream;
    cudaStream_t capture_stream = nullptr;
    std::vector<GraphSlot> graphs;
};

static inline uint32_t rd32(const uint8_t* p) { uint32_t v; memcpy(&v, p, 4); return v; }
static inline uint64_t rd64(const uint8_t* p) { uint64_t v; memcpy(&v, p, 8); return v; }
static inline size_t up256(size_t x) { return (x + 255) & ~(size_t)255; }

extern "C" const char* aceapex_strerror(int code) {
    switch (code) {
        case ACEAPEX_OK: return "ok";
        case ACEAPEX_E_MAGIC: return "bad magic";
        case ACEAPEX_E_VERSION: return "unsupported version";
        case ACEAPEX_E_TRUNCATED: return "compressed buffer truncated";
        case ACEAPEX_E_HEADER: return "inconsistent header or directory";
        case ACEAPEX_E_CAPACITY: return "output or scratch capacity too small";
        case ACEAPEX_E_ALIGN: return "device pointer not 16-byte aligned";
        case ACEAPEX_E_CUDA: return "CUDA runtime error";
        case ACEAPEX_E_ARG: return "bad argument";
        case ACEAPEX_E_STREAM: return "token stream fault detected on the device";
        case ACEAPEX_E_NOMEM: return "host allocation failed";
        case ACEAPEX_E_NOALLOC_LIMIT: return "stream needs more scratch than the library's static no-allocation buffer holds (aceapex_noalloc_max_scratch_bytes)";
        default: return "unknown error";
    }
}

// Wave strategy = the cheapest of four cost estimates built from the header (sequences, matches, blocks, depths with
// matches) and per-unit costs measured on B200 (picoseconds per sequence / match, microseconds per step):
//   PASSES      literal pass 6.1 ps/seq (7.5 when it lists sparse depths) + per dense depth one streaming pass 3.6 ps/seq
//               (+ ~3 us launch) + 8.8 ps per match copied; per sparse depth one list wave (5.5 us + 21 ps per match)
//   LAUNCH      bucketing pass (k_pre) 14.5 ps/seq + per non-empty depth one launch ~5.5 us + 21 ps per match copied from a list
//   PERSISTENT  the same lists, one cooperative kernel: ~3.6 us of grid barrier + fence drain + straggler wait per depth
//   CHAIN       (FLATTENED streams only) literal pass 3.1 ps/seq, then one pass whose time is the larger of the block chain
//               (one ~5.5 us hop per 1 MB block) and its issue-bound throughput (26 ps/seq)
// PASSES is limited to PASS_MAX_DEPTH waves.
static int choose_strategy(const aceapex_plan_t* p) {
    if (p->max_depth == 0) return ACEAPEX_WAVES_LAUNCH;
    double waves = 0;
    for (uint32_t d = 1; d <= p->max_depth; ++d) waves += p->hist_cnt[d] != 0;
    const double seq = (double)p->total_seq, m = (double)p->n_match;
    const double t_lists = 14.5e-6 * seq + 21e-6 * m;                           // microseconds
    const double t_launch = t_lists + 5.5 * waves, t_persist = t_lists + 3.6 * waves + 8.0;
    double t_passes = 1e300;
    if (p->max_depth <= PASS_MAX_DEPTH) {
        t_passes = (p->list_mask ? 7.5e-6 : 6.1e-6) * seq;                     // literal pass (+ listing the sparse depths)
        for (uint32_t d = 1; d <= p->max_depth; ++d)
            t_passes += ((p->list_mask >> d) & 1u) ? 5.5 + 21e-6 * (double)p->hist_cnt[d] : 3.0 + 3.6e-6 * seq + 8.8e-6 * (double)p->hist_cnt[d];
    }
    const double hop = 5.5 * p->n_blocks, thr = 26e-6 * seq;
    const double t_chain = (p->flags & FLAG_FLATTENED) ? 3.1e-6 * seq + (hop > thr ? hop : thr) + 10.0 : 1e300;
    int best = ACEAPEX_WAVES_LAUNCH; double t = t_launch;
    if (t_persist < t) { best = ACEAPEX_WAVES_PERSISTENT; t = t_persist; }
    if (t_passes < t) { best = ACEAPEX_WAVES_PASSES; t = t_passes; }
    if (t_chain < t) { best = ACEAPEX_WAVES_CHAIN; t = t_chain; }
    return best;
}

extern "C" int aceapex_plan(const void* comp_host, size_t comp_bytes, int device, aceapex_plan_t** out) {
    if (!out) return ACEAPEX_E_ARG;
    *out = nullptr;
    if (!comp_host || device < 0) return ACEAPEX_E_ARG;
    const uint8_t* c = static_cast<const uint8_t*>(comp_host);
    if (comp_bytes < HDR_BYTES) return ACEAPEX_E_TRUNCATED;
    if (memcmp(c, "ACEAPEX1", 8) != 0) return ACEAPEX_E_MAGIC;
    if (rd32(c + 8) != 1) return ACEAPEX_E_VERSION;
    aceapex_plan_t* p = new (std::nothrow) aceapex_plan_t();
    if (!p) return ACEAPEX_E_NOMEM;
    int rc = ACEAPEX_OK;
    do {
        p->flags = rd32(c + 12); p->raw_size = rd64(c + 16); p->block_size = rd32(c + 24); p->n_blocks = rd32(c + 28);
        p->min_match = rd32(c + 32); p->depth_limit = rd32(c + 36); p->max_depth = rd32(c + 40);
        p->total_seq = rd64(c + 48); p->total_lit = rd64(c + 56); p->comp_bytes = comp_bytes;
        if (p->block_size == 0 || p->block_size > (1u << 28) || p->raw_size > 0xFFFFFFFFull || p->max_depth > 65535 ||
            p->min_match == 0 || p->total_seq >= 0xFFFFFFF0ull || !(p->flags & FLAG_HAS_DEP)) { rc = ACEAPEX_E_HEADER; break; }
        const uint64_t nb = (p->raw_size + p->block_size - 1) / p->block_size;
        if (nb != p->n_blocks) { rc = ACEAPEX_E_HEADER; break; }
        const uint64_t meta = HDR_BYTES + (uint64_t)DIR_BYTES * nb + (uint64_t)HIST_BYTES * (p->max_depth + 1ull);
        const uint64_t meta_p = (meta + 127) & ~127ull;
        if (meta_p > comp_bytes) { rc = ACEAPEX_E_TRUNCATED; break; }
        const uint8_t* dir = c + HDR_BYTES;
        const uint8_t* hist = dir + DIR_BYTES * nb;
        uint64_t prev_end = meta_p, ts = 0, tl = 0, tiles = 0, tiles_s = 0;
        for (uint64_t b = 0; b < nb && rc == ACEAPEX_OK; ++b) {
            const uint64_t po = rd64(dir + 16 * b); const uint32_t ns = rd32(dir + 16 * b + 8), nl = rd32(dir + 16 * b + 12);
            if ((po & 127) || po < prev_end || ns == 0) { rc = ACEAPEX_E_HEADER; break; }
            const uint64_t bytes = 3 * pad16(2ull * ns) + pad16(4ull * ns) + pad16(nl);
            if (po > comp_bytes || bytes > comp_bytes - po) { rc = ACEAPEX_E_TRUNCATED; break; }
            prev_end = po + bytes; ts += ns; tl += nl; tiles += (ns + TILE_LIST - 1) / TILE_LIST; tiles_s += (ns + TILE_STREAM - 1) / TILE_STREAM;
        }
        if (rc) break;
        if (ts != p->total_seq || tl != p->total_lit || tl > p->raw_size || tiles_s > 0xFFFFFFF0ull) { rc = ACEAPEX_E_HEADER; break; }
        p->n_tiles_list = (uint32_t)tiles; p->n_tiles_stream = (uint32_t)tiles_s;
        p->hist_cnt.resize(p->max_depth + 1); p->hist_bytes.resize(p->max_depth + 1);
        uint64_t nm = 0, mb = 0;
        for (uint32_t d = 0; d <= p->max_depth; ++d) {
            p->hist_cnt[d] = rd32(hist + 16 * d); p->hist_bytes[d] = rd64(hist + 16 * d + 8);
            if (d) { nm += p->hist_cnt[d]; mb += p->hist_bytes[d]; }
        }
        if (nm > p->total_seq || p->hist_bytes[0] != p->total_lit || mb + p->total_lit != p->raw_size ||
            (p->max_depth && p->hist_cnt[p->max_depth] == 0)) { rc = ACEAPEX_E_HEADER; break; }
        p->n_match = nm;
        // device facts
        cudaDeviceProp prop;
        int cur = -1;
        cudaError_t ce = cudaGetDevice(&cur);
        if (ce == cudaSuccess) ce = cudaSetDevice(device);
        if (ce == cudaSuccess) ce = cudaGetDeviceProperties(&prop, device);
        if (ce == cudaSuccess) ce = pre_configure();
        if (ce == cudaSuccess) ce = waves_configure();
        if (ce == cudaSuccess) ce = chain_configure();
        if (ce == cudaSuccess) ce = pass_configure();
        if (ce != cudaSuccess) { p->last_cuda = (int)ce; rc = ACEAPEX_E_CUDA; cudaGetLastError(); break; }
        p->device = device; p->n_sm = prop.multiProcessorCount;
        int pre_occ = pre_max_ctas_per_sm(p->max_depth); if (pre_occ < 1) pre_occ = 1;
        p->pre_grid = p->n_sm * pre_occ;
        { int so = chain_max_ctas_per_sm(); if (so < 1) so = 1; p->chain_grid = p->n_sm * so; }
        { int po = pass_max_ctas_per_sm(); if (po < 1) po = 1; p->pass_grid = p->n_sm * po; }
        p->match_ctas_per_sm = match_max_ctas_per_sm(); if (p->match_ctas_per_sm < 1) p->match_ctas_per_sm = 1;
        if (cur >= 0 && cur != device) cudaSetDevice(cur);
        // scratch layout
        size_t o = 0;
        p->o_status = o; o += up256(sizeof(Status));
        p->o_wave_off = o; o += up256(4ull * (p->max_depth + 2));
        p->o_cursor = o; o += up256(4ull * (p->max_depth + 2));
        p->o_blocks = o; o += up256(sizeof(BlockDesc) * (size_t)nb);
        p->o_tiles = o; o += up256(8ull * p->n_tiles_stream);       // (sized for the finer tiling)
        p->o_tblk = o; o += up256(4ull * p->n_tiles_stream);
        p->o_chain = o; o += up256(4ull * chain_sync_words((uint32_t)nb));
        p->lit_q_cap = (uint32_t)(p->total_lit / LONG_LIT);         // every queued piece is longer than LONG_LIT bytes
        p->o_litq = o; o += up256(16ull * p->lit_q_cap);
        p->o_dst = o; o += up256(4ull * nm);
        p->o_off = o; o += up256(4ull * nm);
        p->o_len = o; o += up256(2ull * nm);
        p->scratch_bytes = o;
        // strategy PASSES: a depth holding fewer than 1/8 of the sequences is cheaper to list in the literal pass and copy
        // from the list (21 ps per match) than to find with a sweep over the whole stream (3.6 ps per sequence)
        p->list_mask = 0;
        if (p->max_depth <= PASS_MAX_DEPTH)
            for (uint32_t d = 1; d <= p->max_depth; ++d)
                if (p->hist_cnt[d] && p->hist_cnt[d] * 8 < p->total_seq) p->list_mask |= 1u << d;
        p->strategy_forced = ACEAPEX_WAVES_AUTO;
        p->strategy_auto = choose_strategy(p);
        p->last_strategy = p->strategy_auto;
    } while (0);
    if (rc) { delete p; return rc; }
    *out = p;
    return ACEAPEX_OK;
}

extern "C" size_t aceapex_raw_bytes(const aceapex_plan_t* p) { return p ? (size_t)p->raw_size : 0; }
extern "C" size_t aceapex_out_bytes(const aceapex_plan_t* p) { return p ? (size_t)((p->raw_size + 15) & ~15ull) : 0; }
extern "C" size_t aceapex_scratch_bytes(const aceapex_plan_t* p) { return p ? p->scratch_bytes : 0; }
extern "C" int aceapex_last_cuda_error(const aceapex_plan_t* p) { return p ? p->last_cuda : 0; }

extern "C" int aceapex_set_strategy(aceapex_plan_t* p, int s) {
    if (!p || s < ACEAPEX_WAVES_AUTO || s > ACEAPEX_WAVES_CHAIN) return ACEAPEX_E_ARG;
    if (s == ACEAPEX_WAVES_PASSES && p->max_depth > PASS_MAX_DEPTH) return ACEAPEX_E_ARG;
    if (s == ACEAPEX_WAVES_CHAIN && !(p->flags & FLAG_FLATTENED)) return ACEAPEX_E_ARG;   // needs invariant I3
    p->strategy_forced = s;
    return ACEAPEX_OK;
}

static Params make_params(const aceapex_plan_t* p, const void* comp_dev, void* out_dev, void* scratch_dev, int strategy) {
    Params P;
    uint8_t* s = static_cast<uint8_t*>(scratch_dev);
    P.comp = static_cast<const uint8_t*>(comp_dev); P.out = static_cast<uint8_t*>(out_dev);
    P.status = reinterpret_cast<Status*>(s + p->o_status);
    P.wave_off = reinterpret_cast<uint32_t*>(s + p->o_wave_off);
    P.cursor = reinterpret_cast<uint32_t*>(s + p->o_cursor);
    P.blocks = reinterpret_cast<BlockDesc*>(s + p->o_blocks);
    P.tile_state = reinterpret_cast<unsigned long long*>(s + p->o_tiles);
    P.tile_blk = reinterpret_cast<uint32_t*>(s + p->o_tblk);
    P.chain_sync = reinterpret_cast<uint32_t*>(s + p->o_chain);
    P.lit_q = reinterpret_cast<uint4*>(s + p->o_litq); P.lit_q_cap = p->lit_q_cap;
    // hist[0] = (literal runs, literal bytes): a mean run of 4-20 bytes means most runs are of the 5-16 byte kind (measured: text
    // MIN 11, mean 12-15 B: literal pass -21 %; stress2g, mean 25 B but bimodal — 1-2 B runs of its text, ~260 B of its random
    // segments: +23 %, so it keeps the byte-loop instance)
    P.long_runs = p->total_lit > 4 * p->hist_cnt[0] && p->total_lit <= 20 * p->hist_cnt[0];
    P.wl_dst = reinterpret_cast<uint32_t*>(s + p->o_dst);
    P.wl_off = reinterpret_cast<uint32_t*>(s + p->o_off);
    P.wl_len = reinterpret_cast<uint16_t*>(s + p->o_len);
    P.raw_size = p->raw_size; P.comp_bytes = p->comp_bytes; P.block_size = p->block_size; P.n_blocks = p->n_blocks;
    const bool stream_tiles = strategy == ACEAPEX_WAVES_PASSES || strategy == ACEAPEX_WAVES_CHAIN;
    P.tile = stream_tiles ? TILE_STREAM : TILE_LIST; P.n_tiles = stream_tiles ? p->n_tiles_stream : p->n_tiles_list; P.max_depth = p->max_depth; P.min_match = p->min_match;
    // strategy CHAIN: no wave list at all (k_chain copies every match straight from the stream, in block order)
    P.list_hi = strategy == ACEAPEX_WAVES_CHAIN ? 0 : p->max_depth;
    P.list_mask = strategy == ACEAPEX_WAVES_PASSES ? p->list_mask : 0;
    uint64_t nl = 0;
    for (uint32_t d = 1; d <= P.list_hi; ++d) nl += p->hist_cnt[d];
    P.n_list = (uint32_t)nl;
    return P;
}

// Enqueue the kernels of one decode on `st`; returns the number of kernel launches through *n_launch.
static cudaError_t enqueue(aceapex_plan_t* p, const Params& P, unsigned phases, int strategy, cudaStream_t st, uint32_t* n_launch) {
    uint32_t n = 0;
    *n_launch = 0;
    if (p->n_blocks == 0) return cudaSuccess;
    const bool chain = strategy == ACEAPEX_WAVES_CHAIN;
    if (strategy == ACEAPEX_WAVES_PASSES) {
        if (phases & ACEAPEX_PHASE_PRE) {
            // short matches are OR-merged into the output (copy.cuh merge16): start from zeros
            if (p->max_depth) {
                cudaError_t ez = cudaMemsetAsync(P.out, 0, (size_t)p->raw_size, st);
                if (ez != cudaSuccess) return ez;
            }
            launch_index(P, st); launch_tilesum(P, p->n_sm * 8, st); launch_pass(P, 0, p->pass_grid, st);
            launch_litcopy(P, p->n_sm * 8, st);
            n += 2 + (P.n_tiles ? 1 : 0) + (P.lit_q_cap ? 1 : 0);
        }
        if ((phases & ACEAPEX_PHASE_MATCH) && p->max_depth) {
            // every depth gets its pass, also one the histogram calls empty: the passes do the token validation
            // (a sparse depth was listed by the literal pass: its matches are copied from the list)
            launch_pass_reset(P, st); ++n;
            for (uint32_t d = 1; d <= p->max_depth; ++d) {
                if ((P.list_mask >> d) & 1u) {
                    cudaError_t e = launch_wave(P, d, (uint32_t)p->hist_cnt[d], p->n_sm * p->match_ctas_per_sm, st);
                    if (e != cudaSuccess) return e;
                    ++n;
                } else { launch_pass(P, d, p->pass_grid, st); n += P.n_tiles ? 1 : 0; }
            }
            launch_check_cursors(P, st); ++n;
        }
        *n_launch = n;
        return cudaGetLastError();
    }
    if (phases & ACEAPEX_PHASE_PRE) {
        // the wave kernel OR-merges short matches into the output (copy.cuh merge16): start from zeros
        if (P.list_hi) {
            cudaError_t ez = cudaMemsetAsync(P.out, 0, (size_t)p->raw_size, st);
            if (ez != cudaSuccess) return ez;
        }
        launch_index(P, st); ++n;
        launch_tilesum(P, p->n_sm * 8, st); ++n;
        if (chain) { launch_pass(P, 0, p->pass_grid, st); n += P.n_tiles ? 1 : 0; }   // literal scatter only: the chain pass validates and counts
        else { launch_pre(P, p->pre_grid, st); n += (P.n_tiles ? 1 : 0) + (P.list_hi ? 1 : 0); }
        launch_litcopy(P, p->n_sm * 8, st); n += P.lit_q_cap ? 1 : 0;
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    if ((phases & ACEAPEX_PHASE_MATCH) && p->max_depth && chain) {
        // one pass over the token stream in block order (replayable: counts, M_src and frontier restart from zero)
        cudaError_t e = cudaMemsetAsync(&P.status->match_src_bytes, 0, sizeof(unsigned long long) + sizeof(uint32_t), st);
        if (e == cudaSuccess) e = launch_chain(P, p->chain_grid, st);
        if (e != cudaSuccess) return e;
        n += P.n_tiles ? 1 : 0;
    } else if ((phases & ACEAPEX_PHASE_MATCH) && p->max_depth) {
        const int wave_grid = p->n_sm * p->match_ctas_per_sm;
        if (strategy == ACEAPEX_WAVES_PERSISTENT) {
            cudaError_t e = launch_waves_persistent(P, 1, P.list_hi, wave_grid, st);
            if (e != cudaSuccess) return e;
            ++n;
        } else {
            for (uint32_t d = 1; d <= P.list_hi; ++d) {
                cudaError_t e = launch_wave(P, d, (uint32_t)p->hist_cnt[d], wave_grid, st);
                if (e != cudaSuccess) return e;
                if (p->hist_cnt[d]) ++n;
            }
        }
    }
    *n_launch = n;
    return cudaGetLastError();
}

extern "C" int aceapex_decode(aceapex_plan_t* p, const void* comp_dev, void* out_dev, size_t out_capacity,
                              void* scratch_dev, size_t scratch_bytes, unsigned phases, void* stream) {
    if (!p || !(phases & ACEAPEX_PHASE_ALL) || (phases & ~(unsigned)ACEAPEX_PHASE_ALL)) return ACEAPEX_E_ARG;
    if (p->n_blocks == 0) { p->last_launches = 0; p->last_stream = (cudaStream_t)stream; return ACEAPEX_OK; }
    if (!comp_dev || !out_dev || !scratch_dev) return ACEAPEX_E_ARG;
    if (out_capacity < aceapex_out_bytes(p) || scratch_bytes < p->scratch_bytes) return ACEAPEX_E_CAPACITY;
    if (((uintptr_t)comp_dev | (uintptr_t)out_dev | (uintptr_t)scratch_dev) & 15) return ACEAPEX_E_ALIGN;
    cudaStream_t st = (cudaStream_t)stream;
    cudaError_t e;
    {   // kernel attributes and grid sizes were set up for the plan's device: refuse to launch anywhere else
        int cur = -1;
        e = cudaGetDevice(&cur);
        if (e != cudaSuccess) { p->last_cuda = (int)e; return ACEAPEX_E_CUDA; }
        if (cur != p->device) return ACEAPEX_E_ARG;
    }
    p->last_stream = st;
    const int strategy = p->strategy_forced != ACEAPEX_WAVES_AUTO ? p->strategy_forced : p->strategy_auto;
    p->last_strategy = strategy;
    p->last_had_match = (phases & ACEAPEX_PHASE_MATCH) != 0;
    const Params P = make_params(p, comp_dev, out_dev, scratch_dev, strategy);
    if (strategy != ACEAPEX_WAVES_GRAPH) {
        e = enqueue(p, P, phases, strategy, st, &p->last_launches);
        if (e != cudaSuccess) { p->last_cuda = (int)e; return ACEAPEX_E_CUDA; }
        return ACEAPEX_OK;
    }
    // ---- CUDA graph: the launch sequence depends only on the plan and the three pointers; cache it
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(st, &cs) == cudaSuccess && cs != cudaStreamCaptureStatusNone) {   // caller is capturing already
        e = enqueue(p, P, phases, ACEAPEX_WAVES_LAUNCH, st, &p->last_launches);
        if (e != cudaSuccess) { p->last_cuda = (int)e; return ACEAPEX_E_CUDA; }
        return ACEAPEX_OK;
    }
    for (GraphSlot& g : p->graphs)
        if (g.comp == comp_dev && g.out == out_dev && g.scratch == scratch_dev && g.phases == phases) {
            e = cudaGraphLaunch(g.exec, st);
            if (e != cudaSuccess) { p->last_cuda = (int)e; return ACEAPEX_E_CUDA; }
            p->last_launches = g.n_launches;
            return ACEAPEX_OK;
        }
    // Capture on a private stream (the caller's may be the legacy default stream, which cannot be captured);
    // capturing records the launches without running them, the instantiated graph then runs on the caller's stream.
    cudaGraph_t graph = nullptr; cudaGraphExec_t exec = nullptr; uint32_t nl = 0;
    e = cudaSuccess;
    if (!p->capture_stream) e = cudaStreamCreateWithFlags(&p->capture_stream, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaStreamBeginCapture(p->capture_stream, cudaStreamCaptureModeThreadLocal);
    if (e == cudaSuccess) {
        cudaError_t e2 = enqueue(p, P, phases, ACEAPEX_WAVES_LAUNCH, p->capture_stream, &nl);
        e = cudaStreamEndCapture(p->capture_stream, &graph);
        if (e2 != cudaSuccess) e = e2;
    }
    if (e == cudaSuccess) e = cudaGraphInstantiate(&exec, graph, 0);
    if (graph) cudaGraphDestroy(graph);
    if (e == cudaSuccess) e = cudaGraphLaunch(exec, st);
    if (e != cudaSuccess) { if (exec) cudaGraphExecDestroy(exec); p->last_cuda = (int)e; cudaGetLastError(); return ACEAPEX_E_CUDA; }
    if (p->graphs.size() >= 8) { cudaGraphExecDestroy(p->graphs.front().exec); p->graphs.erase(p->graphs.begin()); }
    p->graphs.push_back(GraphSlot{comp_dev, out_dev, scratch_dev, phases, strategy, exec, nl});
    p->last_launches = nl;
    return ACEAPEX_OK;
}

extern "C" int aceapex_decode_host(aceapex_plan_t* p, const void* comp_host, size_t comp_bytes, void* out_host,
                                   size_t out_host_capacity, void* comp_dev, void* out_dev, size_t out_capacity,
                                   void* scratch_dev, size_t scratch_bytes, void* stream) {
    if (!p || !comp_host || (!out_host && p->raw_size)) return ACEAPEX_E_ARG;
    if (comp_bytes != p->comp_bytes) return ACEAPEX_E_ARG;
    if (out_host_capacity < p->raw_size) return ACEAPEX_E_CAPACITY;
    if (p->n_blocks == 0) return ACEAPEX_OK;
    if (!comp_dev) return ACEAPEX_E_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    cudaError_t e = cudaMemcpyAsync(comp_dev, comp_host, comp_bytes, cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) { p->last_cuda = (int)e; return ACEAPEX_E_CUDA; }
    int rc = aceapex_decode(p, comp_dev, out_dev, out_capacity, scratch_dev, scratch_bytes, ACEAPEX_PHASE_ALL, stream);
    if (rc) return rc;
    e = cudaMemcpyAsync(out_host, out_dev, p->raw_size, cudaMemcpyDeviceToHost, st);
    if (e != cudaSuccess) { p->last_cuda = (int)e; return ACEAPEX_E_CUDA; }
    return ACEAPEX_OK;
}

extern "C" int aceapex_get_stats(aceapex_plan_t* p, const void* scratch_dev, aceapex_stats* s) {
    if (!p || !s) return ACEAPEX_E_ARG;
    memset(s, 0, sizeof *s);
    s->raw_bytes = p->raw_size; s->comp_bytes = p->comp_bytes; s->lit_bytes = p->total_lit;
    s->match_bytes = p->raw_size - p->total_lit; s->n_seq = p->total_seq; s->n_match = p->n_match;
    s->n_blocks = p->n_blocks; s->block_size = p->block_size; s->min_match = p->min_match; s->max_depth = p->max_depth;
    s->depth_limit = p->depth_limit; s->flags = p->flags; s->strategy = (uint32_t)p->last_strategy;
    s->n_launches = p->last_launches;
    if (scratch_dev && p->n_blocks) {
        Status h;
        cudaError_t e = cudaStreamSynchronize(p->last_stream);
        if (e == cudaSuccess) e = cudaMemcpy(&h, static_cast<const uint8_t*>(scratch_dev) + p->o_status, sizeof h, cudaMemcpyDeviceToHost);
        if (e != cudaSuccess) { p->last_cuda = (int)e; return ACEAPEX_E_CUDA; }
        s->match_src_bytes = h.match_src_bytes + h.src_bytes_pre; s->fault_flags = h.fault_flags; s->fault_block = h.fault_block;
        // strategy CHAIN keeps no list (hence no cursor): its match count comes back from the chain pass
        if (!h.fault_flags && p->last_strategy == ACEAPEX_WAVES_CHAIN && p->max_depth && p->last_had_match && h.n_final != p->n_match) {
            s->fault_flags = F_DEPTH; s->fault_block = 0xFFFFFFFEu;
        }
        if (s->fault_flags) return ACEAPEX_E_STREAM;
    }
    return ACEAPEX_OK;
}

extern "C" int64_t aceapex_depth_hist(const aceapex_plan_t* p, uint64_t* n_match, uint64_t* n_bytes, uint32_t cap) {
    if (!p) return ACEAPEX_E_ARG;
    for (uint32_t d = 0; d <= p->max_depth && d < cap; ++d) {
        if (n_match) n_match[d] = p->hist_cnt[d];
        if (n_bytes) n_bytes[d] = p->hist_bytes[d];
    }
    return (int64_t)p->max_depth + 1;
}

extern "C" void aceapex_free(aceapex_plan_t* p) {
    if (!p) return;
    for (GraphSlot& g : p->graphs) cudaGraphExecDestroy(g.exec);
    if (p->capture_stream) cudaStreamDestroy(p->capture_stream);
    delete p;
}

// ---------------------------------------------------------------------------------------------------------------------
// No-allocation entry point (include/aceapex.h: aceapex_decode_noalloc).  For callers that cannot obtain device scratch
// (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc): the same kernels, with their
// scratch (status words, block descriptors, tile prefixes, wave lists, literal queue, chain counters — the layout of
// aceapex_scratch_bytes) placed in ONE file-scope device array owned by the library.  NOALLOC_MAX bytes are held by every
// GPU that loads the library, until the process exits.  Nothing here calls cudaMalloc / cudaFree / an allocating routine
// (strategy GRAPH, which instantiates a graph, is run as LAUNCH).
//  * In host code the array's NAME is a host-side stand-in, not a device address: the address comes from
//    cudaGetSymbolAddress, once per device, with that device current (noalloc_scratch below), and that pointer is what the
//    kernels get (through Params, like a caller's scratch).
//  * Every call shares the array and finds the previous call's contents in it.  Nothing relies on them: the decode
//    always runs PHASE_PRE, whose first kernel (k_index) resets the status words, cursors and the queue count, and the
//    chain / barrier counters are cleared by the launches that use them — exactly as with a caller's uninitialised scratch.
//  * Calls that overlap on the GPU (two streams, two plans, two host threads) race on the array: one call at a time per
//    device; aceapex_get_stats_noalloc must be called before the next aceapex_decode_noalloc on that device.
namespace {
constexpr size_t NOALLOC_MAX = (size_t)16 << 20;     // 16 MiB: a stream of up to ~1.4 M sequences (config 0, 4 MB, needs 5.6 MB)
constexpr int NOALLOC_MAX_DEVICES = 64;
static __device__ __align__(256) unsigned char ax_noalloc_scratch[NOALLOC_MAX];
std::mutex g_noalloc_mu;
void* g_noalloc_ptr[NOALLOC_MAX_DEVICES];            // device address of ax_noalloc_scratch, per device ordinal (0 = not set up)

// Set-up, once per device, with that device current.
cudaError_t noalloc_scratch(int device, void** out) {
    if (device < 0 || device >= NOALLOC_MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lk(g_noalloc_mu);
    if (!g_noalloc_ptr[device]) {
        void* ptr = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&ptr, ax_noalloc_scratch);
        if (e != cudaSuccess) return e;
        if (!ptr || ((uintptr_t)ptr & 255)) return cudaErrorInvalidSymbol;
        g_noalloc_ptr[device] = ptr;
    }
    *out = g_noalloc_ptr[device];
    return cudaSuccess;
}
}  // namespace

extern "C" size_t aceapex_noalloc_max_scratch_bytes(void) { return NOALLOC_MAX; }

extern "C" int aceapex_decode_noalloc(aceapex_plan_t* p, const void* comp_dev, void* out_dev, size_t out_capacity, void* stream) {
    if (!p) return ACEAPEX_E_ARG;
    if (p->scratch_bytes > NOALLOC_MAX) return ACEAPEX_E_NOALLOC_LIMIT;          // stated maximum: rejected, nothing launched
    if (p->n_blocks == 0) { p->last_launches = 0; p->last_stream = (cudaStream_t)stream; return ACEAPEX_OK; }
    if (!comp_dev || !out_dev) return ACEAPEX_E_ARG;
    if (out_capacity < aceapex_out_bytes(p)) return ACEAPEX_E_CAPACITY;
    if (((uintptr_t)comp_dev | (uintptr_t)out_dev) & 15) return ACEAPEX_E_ALIGN;
    int cur = -1;
    cudaError_t e = cudaGetDevice(&cur);
    if (e != cudaSuccess) { p->last_cuda = (int)e; return ACEAPEX_E_CUDA; }
    if (cur != p->device) return ACEAPEX_E_ARG;                                   // kernel attributes / grids belong to the plan's device
    void* scratch = nullptr;
    e = noalloc_scratch(cur, &scratch);
    if (e != cudaSuccess) { p->last_cuda = (int)e; cudaGetLastError(); return ACEAPEX_E_CUDA; }
    cudaStream_t st = (cudaStream_t)stream;
    int strategy = p->strategy_forced != ACEAPEX_WAVES_AUTO ? p->strategy_forced : p->strategy_auto;
    if (strategy == ACEAPEX_WAVES_GRAPH) strategy = ACEAPEX_WAVES_LAUNCH;        // (instantiating a graph allocates)
    p->last_stream = st; p->last_strategy = strategy; p->last_had_match = true;
    const Params P = make_params(p, comp_dev, out_dev, scratch, strategy);
    e = enqueue(p, P, ACEAPEX_PHASE_ALL, strategy, st, &p->last_launches);
    if (e != cudaSuccess) { p->last_cuda = (int)e; return ACEAPEX_E_CUDA; }
    return ACEAPEX_OK;
}

extern "C" int aceapex_get_stats_noalloc(aceapex_plan_t* p, aceapex_stats* s) {
    if (!p || !s) return ACEAPEX_E_ARG;
    void* scratch = nullptr;
    if (p->n_blocks) {
        int cur = -1;
        cudaError_t e = cudaGetDevice(&cur);
        if (e == cudaSuccess && cur != p->device) return ACEAPEX_E_ARG;
        if (e == cudaSuccess) e = noalloc_scratch(cur, &scratch);
        if (e != cudaSuccess) { p->last_cuda = (int)e; cudaGetLastError(); return ACEAPEX_E_CUDA; }
    }
    return aceapex_get_stats(p, scratch, s);
}
