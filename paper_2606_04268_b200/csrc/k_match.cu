// k_match.cu — steps a6/a7: wavefront match copy, one wave per dependency depth (§4.4: "all
// level-k tokens are processed in parallel"; §7.1: "within each level, tokens are independent").
// Wave d copies, for every match of depth d, len bytes out[off ..) -> out[mdst ..); a source that overlaps
// its destination (mdst - off < len) is the periodic extension of out[off .. mdst) (Q3).
//
// Work assignment: the measured length mix is 98 % <= 16 bytes on the text and FASTQ workloads, so
// one THREAD copies one short match (len <= SHORT_MAX) through registers — the source is read as one or two
// aligned 16-byte words and funnel-shifted, the destination is OR-merged into the zeroed output with 8-byte L2
// reductions (copy.cuh merge16) — and one WARP copies one long match with 16-byte vector stores.
// Sequencing (a7): k_waves runs all depths in one cooperative launch with a grid barrier between
// waves (strategy PERSISTENT), or one depth per ordinary launch (LAUNCH; GRAPH replays those launches from a CUDA
// graph, the paper's mechanism).
// Every source byte of wave d was written by an earlier wave or by the literal scatter.  Loads of `out` are plain
// (L1-cached) loads: a kernel boundary, or the acquiring spin of the grid barrier (CCTL.IVALL), invalidates L1 before any wave
// reads what an earlier wave wrote on another SM.  No store or merge changes a byte outside the match's own range.
#include "common.cuh"
#include "copy.cuh"

namespace ax {

// ---- the wave kernel: a software pipeline over "pieces" of the wave lists
// CTA c owns the slice [first + c*per, first + (c+1)*per) of every wave's list, cut into pieces of <= PIECE
// entries.  Stage k+2's entries travel global -> shared with cp.async (no registers, no stall) while stage k+1's
// destination lines are prefetched into L2 (the OR-merge is a read-modify-write there) and stage k is copied, so
// after a grid barrier only the source loads and the merges themselves are on the critical path (DRAM latency on B200 is ~1 us; a wave costs ~3 of them if the
// entry load, the source load and the barrier are taken one after the other).
constexpr uint32_t PIECE = 4 * PERSIST_THREADS;          // entries per piece (4 per thread)
constexpr uint32_t NSTAGE = 3;
constexpr uint32_t OFF_WIN = 1024;                       // wave_off window kept in shared memory

struct WaveSmem {
    uint32_t dst[NSTAGE][PIECE];
    uint32_t off[NSTAGE][PIECE];
    uint16_t len[NSTAGE][PIECE + 8];
    uint32_t woff[OFF_WIN + 2];
};

struct Piece { uint32_t a, n, depth; bool first_of_wave, valid; };

__device__ __forceinline__ void cp_async4(void* smem, const void* gmem) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"((uint32_t)__cvta_generic_to_shared(smem)), "l"(gmem) : "memory");
}

__global__ void __launch_bounds__(PERSIST_THREADS, 1024 / PERSIST_THREADS) k_waves(Params P, uint32_t d_first, uint32_t d_last) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    WaveSmem& S = *reinterpret_cast<WaveSmem*>(smem_raw);
    if (P.status->fault_flags & F_DEPTH) return;          // wave lists incomplete (k_check_cursors): copy nothing.
                                                          // Uniform over the grid: the flag is final before this kernel starts.
    const uint32_t tid = threadIdx.x, lane = tid & 31, nct = gridDim.x, cta = blockIdx.x;
    // ---- piece iterator (identical in every thread of the CTA)
    uint32_t it_d = d_first, it_pos = 0, it_hi = 0, win0 = d_first;
    bool it_new = true;                                   // the next piece opens wave it_d
    auto load_window = [&]() {
        for (uint32_t i = tid; i < OFF_WIN + 2 && win0 + i <= P.max_depth + 1; i += PERSIST_THREADS) S.woff[i] = P.wave_off[win0 + i];
        __syncthreads();
    };
    load_window();
    auto next_piece = [&]() -> Piece {
        Piece pc; pc.valid = false; pc.a = 0; pc.n = 0; pc.depth = 0; pc.first_of_wave = false;
        if (it_d > d_last) return pc;
        if (it_new) {
            if (it_d - win0 >= OFF_WIN) { __syncthreads(); win0 = it_d; load_window(); }
            const uint32_t first = S.woff[it_d - win0], cnt = S.woff[it_d - win0 + 1] - first;
            const uint32_t per = (cnt + nct - 1) / nct;
            const uint32_t lo = cta * per < cnt ? cta * per : cnt, hi = (cta + 1) * per < cnt ? (cta + 1) * per : cnt;
            it_pos = first + lo; it_hi = first + hi;
        }
        pc.valid = true; pc.depth = it_d; pc.first_of_wave = it_new;
        pc.a = it_pos; pc.n = it_hi - it_pos < PIECE ? it_hi - it_pos : PIECE;
        it_pos += pc.n; it_new = false;
        if (it_pos >= it_hi) { ++it_d; it_new = true; }
        return pc;
    };
    // cp.async the piece's entries into stage st.  `wtid`/`wn`: index and number of the threads that take part (the
    // whole CTA in the prologue; warps 1..31 in the loop, where warp 0 runs the grid barrier at the same time).
    auto issue = [&](const Piece& pc, uint32_t st, uint32_t wtid, uint32_t wn) {
        if (pc.valid) {
            for (uint32_t i = wtid; i < pc.n; i += wn) {
                cp_async4(&S.dst[st][i], P.wl_dst + pc.a + i);
                cp_async4(&S.off[st][i], P.wl_off + pc.a + i);
            }
            // lengths are u16: copy the 4-byte words that cover [a, a+n); S.len[st][i - (a & ~1)] holds entry i
            const uint32_t a2 = pc.a & ~1u, nw = (pc.a + pc.n - a2 + 1) >> 1;
            for (uint32_t w = wtid; w < nw; w += wn) cp_async4(&S.len[st][2 * w], P.wl_len + a2 + 2 * w);
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    // process one landed piece from stage st: rounds of one entry per thread (measured: a single copy_ents<1> body
    // looped beats the 2- and 4-entry unrolled bodies — text256m match phase 1.80 -> 1.73 ms — and is a third of the code)
    auto process = [&](const Piece& cur, uint32_t st) {
        const uint32_t sh = cur.a & 1u;
        for (uint32_t r0 = 0; r0 < cur.n; r0 += PERSIST_THREADS) {
            Ent e[1];
            const uint32_t i = tid + r0;
            e[0].mdst = 0; e[0].off = 0; e[0].len = 0;
            if (i < cur.n) { e[0].mdst = S.dst[st][i]; e[0].off = S.off[st][i]; e[0].len = S.len[st][i + sh]; }
            copy_ents<1>(P.out, e, lane);
        }
    };
    Piece pc[NSTAGE];
    pc[0] = next_piece(); issue(pc[0], 0, tid, PERSIST_THREADS);
    pc[1] = next_piece(); issue(pc[1], 1, tid, PERSIST_THREADS);
    asm volatile("cp.async.wait_group 1;" ::: "memory");   // piece 0 landed (this thread's part)
    __syncthreads();
    uint32_t epoch = 0;
    constexpr uint32_t NW = PERSIST_THREADS - 32;          // threads of warps 1..31
    for (uint32_t k = 0; pc[k % NSTAGE].valid; ++k) {
        const uint32_t s0 = k % NSTAGE, s1 = (k + 1) % NSTAGE, s2 = (k + 2) % NSTAGE;
        const Piece cur = pc[s0];
        process(cur, s0);
        __syncthreads();                                   // every store of this piece is issued; stage s0 is free
        const Piece nxt = pc[s1];
        const bool boundary = nxt.valid && nxt.first_of_wave;   // a7: the next piece opens a new wave
        if (boundary) epoch += nct;
        pc[s2] = next_piece();                             // (uniform bookkeeping, all threads)
        if (tid < 32) {
            // warp 0: the grid barrier (monotone counter in scratch, zeroed before the launch; the cooperative launch
            // guarantees all CTAs are resident) — arrive (release: the CTA's stores are ordered before it through the
            // __syncthreads above), acquiring spin (also invalidates L1: CCTL.IVALL)
            if (boundary && tid == 0) {
                asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(&P.status->barrier), "r"(1u) : "memory");
                uint32_t v;
                // the spin is itself the acquire (LDG.STRONG.GPU + CCTL.IVALL): a relaxed spin + fence.acq_rel.gpu adds a
                // MEMBAR.ALL.GPU per wave (measured 6.84 vs 6.40 ms over the 1024 waves of fastq1g)
                do { asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(&P.status->barrier) : "memory"); } while (v < epoch);
            }
            asm volatile("cp.async.commit_group;" ::: "memory");   // keep every thread's group count in step
            asm volatile("cp.async.wait_group 1;" ::: "memory");   // (warp 0 took part in the prologue's pieces 0 and 1)
        } else {
            // warps 1..31, meanwhile: fetch piece k+2, and once piece k+1 has landed pull the next wave's destination
            // lines into L2 (prefetching the sources too was measured slower: DESIGN.md 6.2)
            issue(pc[s2], s2, tid - 32, NW);
            asm volatile("cp.async.wait_group 1;" ::: "memory");   // piece k+1 landed (this thread's part)
            asm volatile("bar.sync 1, %0;" ::"n"(NW) : "memory");
            if (boundary && k != 0) {                      // (k == 0: piece 1 was issued by all 32 warps, warp 0's part may not have landed)
                const uint32_t sh = nxt.a & 1u;
                for (uint32_t i = tid - 32; i < nxt.n; i += NW)
                    if (S.len[s1][i + sh]) asm volatile("prefetch.global.L2 [%0];" ::"l"(P.out + S.dst[s1][i]));
            }
        }
        __syncthreads();
    }
}

size_t waves_smem_bytes() { return sizeof(WaveSmem); }

cudaError_t waves_configure() {
    return cudaFuncSetAttribute(k_waves, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(WaveSmem));
}

int match_max_ctas_per_sm() {
    int n = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k_waves, PERSIST_THREADS, sizeof(WaveSmem)) != cudaSuccess) return 0;
    return n;
}

// One wave as an ordinary launch (strategies LAUNCH and GRAPH): no barrier is executed when d_first == d_last.
cudaError_t launch_wave(const Params& P, uint32_t depth, uint32_t n_entries, int max_grid, cudaStream_t st) {
    if (n_entries == 0) return cudaSuccess;
    uint32_t grid = (n_entries + PERSIST_THREADS - 1) / PERSIST_THREADS;
    if (grid > (uint32_t)max_grid) grid = max_grid;
    k_waves<<<grid, PERSIST_THREADS, sizeof(WaveSmem), st>>>(P, depth, depth);
    return cudaGetLastError();
}

// All waves d_first .. d_last in one cooperative launch (strategy PERSISTENT).
cudaError_t launch_waves_persistent(const Params& P, uint32_t d_first, uint32_t d_last, int grid, cudaStream_t st) {
    cudaError_t e = cudaMemsetAsync(&P.status->barrier, 0, sizeof(uint32_t), st);
    if (e != cudaSuccess) return e;
    Params p = P;
    void* args[] = {&p, &d_first, &d_last};
    return cudaLaunchCooperativeKernel((const void*)k_waves, dim3(grid), dim3(PERSIST_THREADS), args, sizeof(WaveSmem), st);
}

}  // namespace ax
