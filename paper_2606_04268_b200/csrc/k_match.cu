// k_match.cu — steps a6/a7: wavefront match copy, one wave per dependency depth (§4.4: "all
// level-k tokens are processed in parallel"; §7.1: "within each level, tokens are independent").
// Wave d copies, for every match of depth d, len bytes out[off ..) -> out[mdst ..); a source that overlaps
// its destination (mdst - off < len) is the periodic extension of out[off .. mdst) (Q3).
// Two ways of sequencing the waves (a7): one launch per depth (k_wave; plain or replayed from a CUDA graph,
// PAPER.md:97), or one cooperative kernel with a grid barrier between depths (k_waves_persistent).
// Every source byte of wave d was written by an earlier wave / the literal scatter; loads of `out` bypass L1
// (ld.global.cg) because in the persistent kernel they may have been written by another SM in this launch.
// Stores never touch a byte outside the match's own output range.
#include "common.cuh"

namespace ax {

// One thread copies one short match (len <= SHORT_MAX).
__device__ __forceinline__ void thread_copy(uint8_t* out, uint32_t mdst, uint32_t off, uint32_t len) {
    const uint32_t dist = mdst - off;
    const uint8_t* s = out + off;
    uint8_t* d = out + mdst;
    uint32_t j = 0;
    for (uint32_t i = 0; i < len; ++i) {
        d[i] = __ldcg(s + j);
        if (++j == dist) j = 0;
    }
}

// The matches [first, last) of one wave list, 32 per warp step.
__device__ __forceinline__ void wave_body(const Params& P, uint32_t first, uint32_t last, uint32_t warp_global,
                                          uint32_t n_warps, uint32_t lane) {
    for (uint32_t base = first + warp_global * 32u; base < last; base += n_warps * 32u) {
        const uint32_t i = base + lane;
        uint32_t mdst = 0, off = 0, len = 0;
        if (i < last) { mdst = P.wl_dst[i]; off = P.wl_off[i]; len = P.wl_len[i]; }
        if (len != 0 && len <= SHORT_MAX) thread_copy(P.out, mdst, off, len);
        uint32_t longm = __ballot_sync(0xFFFFFFFFu, len > SHORT_MAX);
        while (longm) {
            const int sl = __ffs(longm) - 1; longm &= longm - 1;
            const uint32_t d2 = __shfl_sync(0xFFFFFFFFu, mdst, sl), o2 = __shfl_sync(0xFFFFFFFFu, off, sl),
                           n2 = __shfl_sync(0xFFFFFFFFu, len, sl);
            const uint32_t dist = d2 - o2;
            if (dist >= n2) warp_copy(P.out + d2, P.out + o2, n2, lane);
            else warp_fill_periodic(P.out + d2, P.out + o2, n2, dist, lane);
        }
    }
}

__device__ __forceinline__ void wave_bounds(const Params& P, uint32_t d, uint32_t& first, uint32_t& last) {
    first = P.wave_off[d];
    const uint32_t cap = P.wave_off[d + 1], cur = P.cursor[d];   // entries actually written by PRE: [first, min(cur, cap))
    last = cur < cap ? cur : cap;
}

__global__ void __launch_bounds__(MATCH_THREADS) k_wave(Params P, uint32_t depth) {
    uint32_t first, last;
    wave_bounds(P, depth, first, last);
    const uint32_t wpb = MATCH_THREADS / 32;
    wave_body(P, first, last, blockIdx.x * wpb + (threadIdx.x >> 5), gridDim.x * wpb, threadIdx.x & 31);
}

// Grid barrier: monotone counter in scratch (zeroed by the host before the launch); cooperative launch
// guarantees all CTAs are resident.  Release: fence before the arrive; acquire: fence after the spin.
__device__ __forceinline__ void grid_barrier(uint32_t* ctr, uint32_t target) {
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        atomicAdd(ctr, 1u);
        uint32_t v;
        do { asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(ctr) : "memory"); } while (v < target);
        __threadfence();
    }
    __syncthreads();
}

__global__ void __launch_bounds__(MATCH_THREADS) k_waves_persistent(Params P, uint32_t d_first, uint32_t d_last) {
    const uint32_t wpb = MATCH_THREADS / 32;
    const uint32_t warp_global = blockIdx.x * wpb + (threadIdx.x >> 5), n_warps = gridDim.x * wpb, lane = threadIdx.x & 31;
    uint32_t epoch = 0;
    for (uint32_t d = d_first; d <= d_last; ++d) {
        uint32_t first, last;
        wave_bounds(P, d, first, last);
        wave_body(P, first, last, warp_global, n_warps, lane);
        if (d != d_last) { epoch += gridDim.x; grid_barrier(&P.status->barrier, epoch); }
    }
}

int match_max_ctas_per_sm() {
    int n = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k_waves_persistent, MATCH_THREADS, 0) != cudaSuccess) return 0;
    return n;
}

cudaError_t launch_wave(const Params& P, uint32_t depth, uint32_t n_entries, int max_grid, cudaStream_t st) {
    if (n_entries == 0) return cudaSuccess;
    uint32_t grid = (n_entries + MATCH_THREADS - 1) / MATCH_THREADS;      // one entry per thread ...
    if (grid > (uint32_t)max_grid) grid = max_grid;                       // ... capped; the warp loop strides
    k_wave<<<grid, MATCH_THREADS, 0, st>>>(P, depth);
    return cudaGetLastError();
}

cudaError_t launch_waves_persistent(const Params& P, uint32_t d_first, uint32_t d_last, int grid, cudaStream_t st) {
    cudaError_t e = cudaMemsetAsync(&P.status->barrier, 0, sizeof(uint32_t), st);
    if (e != cudaSuccess) return e;
    Params p = P;
    void* args[] = {&p, &d_first, &d_last};
    return cudaLaunchCooperativeKernel((const void*)k_waves_persistent, dim3(grid), dim3(MATCH_THREADS), args, 0, st);
}

}  // namespace ax
