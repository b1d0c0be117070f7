// Ranking by a per-pixel bitmap: a set of distinct pixel positions g (one bit each, counted into blocks of 4096
// positions) is ranked in ascending order of g without a sort: rank(g) = exclusive prefix of g's block + popcount of the
// block's bitmap words below g.  Shared by K5 (catalogue slots of detect_sources), K9 (deblended catalogue) and K10
// (compaction after cleaning).  Include inside the file's anonymous namespace.
#pragma once

constexpr int RB_SHIFT = 12;   // ranking blocks of 4096 pixels (128 bitmap words)

// K5s: exclusive scan of the block counts (one CTA; thread t owns a contiguous chunk, held in registers when
// the chunk is <= 32 counts), total -> *total_out.  cnt[] is readable up to the next multiple of 4 past n.
__global__ void __launch_bounds__(1024) k5s_scan_blocks(const uint32_t *cnt, size_t n, uint32_t *prefix, uint32_t *total_out) {
    __shared__ uint32_t red[32];
    bd_pdl_wait();      // (no-ops unless the kernel was launched programmatically dependent)
    bd_pdl_trigger();
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const size_t per = (((n + 1023) / 1024) + 3) & ~(size_t)3, i0 = (size_t)tid * per, i1 = i0 + per < n ? i0 + per : n;
    const bool in_regs = per <= 32;
    uint4 v[8];
    uint32_t local = 0;
    if (in_regs) {
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            v[k] = make_uint4(0, 0, 0, 0);
            const size_t i = i0 + 4 * k;
            if (4 * k < (int)per && i < n) {
                v[k] = *reinterpret_cast<const uint4 *>(cnt + i);
                if (i + 1 >= n) v[k].y = 0;
                if (i + 2 >= n) v[k].z = 0;
                if (i + 3 >= n) v[k].w = 0;
            }
            local += v[k].x + v[k].y + v[k].z + v[k].w;
        }
    } else {
        for (size_t i = i0; i < i1; ++i) local += cnt[i];
    }
    uint32_t incl = local;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { uint32_t t = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += t; }
    if (lane == 31) red[warp] = incl;
    __syncthreads();
    uint32_t run = incl - local, tot = 0;
    for (int w = 0; w < 32; ++w) { if (w < warp) run += red[w]; tot += red[w]; }
    if (in_regs) {
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const size_t i = i0 + 4 * k;
            if (4 * k < (int)per && i < n) {
                uint4 o;
                o.x = run; run += v[k].x; o.y = run; run += v[k].y; o.z = run; run += v[k].z; o.w = run; run += v[k].w;
                *reinterpret_cast<uint4 *>(prefix + i) = o;   // prefix[] has room up to the next multiple of 4 past n + 1
            }
        }
    } else {
        for (size_t i = i0; i < i1; ++i) { const uint32_t c = cnt[i]; prefix[i] = run; run += c; }
    }
    __syncthreads();
    if (tid == 0) { prefix[n] = tot; *total_out = tot; }
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

