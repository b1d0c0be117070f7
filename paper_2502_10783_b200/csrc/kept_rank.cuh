// Ranking by a per-pixel bitmap: a set of distinct pixel positions g (one bit each, counted into blocks of 4096
// positions) is ranked in ascending order of g without a sort: rank(g) = exclusive prefix of g's block + popcount of the
// block's bitmap words below g.  Shared by K5 (catalogue slots of detect_sources), K9 (deblended catalogue) and K10
// (compaction after cleaning).  Include inside the file's anonymous namespace.
#pragma once

constexpr int RB_SHIFT = 12;   // ranking blocks of 4096 pixels (128 bitmap words)

// K5s: exclusive scan of the block counts, total -> *total_out.  One CTA walks the array in tiles of 4096 counts: coalesced
// 128-bit loads, a shuffle scan per warp, the 32 warp totals through shared memory, a running carry, coalesced 128-bit stores.
// (The first version gave every thread one contiguous chunk: fine while a chunk was <= 32 counts held in registers, but the
// 65 536 blocks of config 4 and the 83 k cells of K10 on config 3 took its scalar path with a 256-byte stride between
// neighbouring threads: 121 us.)  cnt[] is readable and prefix[] writable up to the next multiple of 4 past n (+ 1).
__global__ void __launch_bounds__(1024) k5s_scan_blocks(const uint32_t *cnt, size_t n, uint32_t *prefix, uint32_t *total_out) {
    __shared__ uint32_t red[32];
    bd_pdl_wait();      // (no-ops unless the kernel was launched programmatically dependent)
    bd_pdl_trigger();
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    uint32_t carry = 0;
    for (size_t base = 0; base < n; base += 4096) {
        const size_t i = base + 4 * (size_t)tid;
        uint4 v = make_uint4(0, 0, 0, 0);
        if (i < n) {
            v = *reinterpret_cast<const uint4 *>(cnt + i);
            if (i + 1 >= n) v.y = 0;
            if (i + 2 >= n) v.z = 0;
            if (i + 3 >= n) v.w = 0;
        }
        const uint32_t local = v.x + v.y + v.z + v.w;
        uint32_t incl = local;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const uint32_t t = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += t; }
        if (lane == 31) red[warp] = incl;
        __syncthreads();
        uint32_t mine = red[lane], wincl = mine;   // every warp scans the 32 warp totals itself
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const uint32_t t = __shfl_up_sync(0xffffffffu, wincl, o); if (lane >= o) wincl += t; }
        const uint32_t wbase = __shfl_sync(0xffffffffu, wincl - mine, warp), tot = __shfl_sync(0xffffffffu, wincl, 31);
        if (i < n) {
            uint4 o;
            uint32_t run = carry + wbase + incl - local;
            o.x = run; run += v.x; o.y = run; run += v.y; o.z = run; run += v.z; o.w = run;
            *reinterpret_cast<uint4 *>(prefix + i) = o;
        }
        carry += tot;
        __syncthreads();
    }
    if (tid == 0) { prefix[n] = carry; *total_out = carry; }
}

// number of kept roots with global pixel index < g: block prefix + popcount of the block's bitmap words below g
// (<= 128 words, read as predicated 128-bit loads that are all in flight together)
__device__ __forceinline__ uint32_t kept_rank(const uint32_t *keptbits, const uint32_t *blkprefix, size_t g) {
    const size_t w0 = (g >> RB_SHIFT) << (RB_SHIFT - 5);
    const int nw = (int)((g >> 5) - w0);                    // full words below g's word
    const uint32_t pm = (1u << (g & 31)) - 1u;              // partial mask of g's word
    const uint4 *kb = reinterpret_cast<const uint4 *>(keptbits + w0);
    uint32_t rank = __ldg(blkprefix + (g >> RB_SHIFT));
#pragma unroll
    for (int k = 0; k < 32; ++k) {
        if (4 * k <= nw) {
            const uint4 v = __ldg(kb + k);
            const int b = 4 * k;
            rank += __popc(v.x & (b < nw ? 0xFFFFFFFFu : pm));
            rank += __popc(v.y & (b + 1 < nw ? 0xFFFFFFFFu : (b + 1 == nw ? pm : 0u)));
            rank += __popc(v.z & (b + 2 < nw ? 0xFFFFFFFFu : (b + 2 == nw ? pm : 0u)));
            rank += __popc(v.w & (b + 3 < nw ? 0xFFFFFFFFu : (b + 3 == nw ? pm : 0u)));
        }
    }
    return rank;
}

