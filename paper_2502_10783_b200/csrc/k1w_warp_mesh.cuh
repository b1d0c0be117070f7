// K1W: sigma-clipped statistics of SMALL meshes (<= 4096 pixels, mesh_w % 4 == 0: the paper's default 64x64 sub-regions,
// PAPER.md:67), one WARP per mesh, no block barrier anywhere.  Included by k1_mesh_stats.cu (inside its namespace).
//
// The CTA-per-mesh kernel spends 60 of its 68 k cycles per 64x64 mesh in serial phases behind block barriers (sample
// sort, candidate sort, clipping rounds) with 128 threads mostly idle; config 4 (65 536 meshes) took 3.0 ms for a 0.16 ms
// HBM floor.  Here a CTA is one warp: the mesh arrives in shared memory with ONE TMA bulk-tensor load (16 KiB), and the
// warp runs the same two-level scheme as the fast path of k1_mesh_stats with warp shuffles only:
//   sample   256 lattice pixels of the slab, bitonic-sorted in registers (8 keys per lane) -> pivot q50, core interval
//            [A, B] = q50 -+ 2 (q50 - q16) that every clipping bound stays outside of, key bracket [ka, kb] around the median;
//   sweep    ONE pass over the slab: float64 core sums, the count below the bracket, and an IN-PLACE compacted list L of the
//            "interesting" pixels -- tail pixels (outside the core) and bracket candidates -- written over the part of the
//            slab that has already been read (the list can never overtake the read position), so no list has a capacity;
//   window   64-bin histogram of the candidates in L (per-lane byte columns, dp4a), a window of bins around the median rank
//            with <= 256 keys, gathered and sorted in registers: every round's median is then a table lookup;
//   rounds   the tail entries of L are compacted in place once more; each clipping round is one pass of the warp over them
//            (n = n_core + #tail in [lo, hi], sums likewise) and one shuffle reduction.
// A mesh whose assumptions fail (degenerate sample, median rank outside the window, a bound enters the core), or that holds
// fewer than 1024 valid pixels (partial edge meshes), is appended to a worklist that the general kernel serves afterwards.
// float64 sums against float64 bounds: the survivor sets are the float64 definition's (n_kept / median bit-exact).
#pragma once

constexpr int KW_SLAB_BYTES = 16384;      // 4096 pixels
constexpr int KW_WIN = 256;               // window keys (8 per lane)
constexpr int KW_MIN_PX = 1024;           // smaller (edge) meshes go to the general kernel
constexpr int KW_SMEM = KW_SLAB_BYTES + 2048 + 256 + 64;   // slab, byte histogram / window, bin totals, mbarrier

struct K1WArgs {
    const float *img;
    int B, H, W, mh, mw, ny, nx;
    int use_tma;
    double k_c;
    int iters, skew_guard;
    double median_factor, mean_factor;
    double *bkg_raw, *rms_raw, *median, *mean;
    int32_t *n_kept;
    uint32_t *fb_count;   // worklist of the general kernel: count, then mesh indices
    uint32_t *fb_list;
};

// shared-memory accesses of the in-place compactions: volatile asm with a memory clobber, so neither the compiler nor
// type-based alias analysis can move a later read of the slab above an earlier write of the list
__device__ __forceinline__ uint4 kw_lds128(uint32_t addr) {
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ uint32_t kw_lds32(uint32_t addr) {
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ void kw_sts32(uint32_t addr, uint32_t v) {
    asm volatile("st.shared.u32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}

__global__ void __launch_bounds__(32) k1w_warp_mesh(const __grid_constant__ CUtensorMap tmap, K1WArgs a) {
    extern __shared__ __align__(128) unsigned char sm[];
    const uint32_t slab_s = smem_u32(sm);                         // the mesh; then list L (keys); then tail list T
    uint8_t *hist8 = sm + KW_SLAB_BYTES;                          // [64][32] byte counters; then the sorted window
    uint32_t *win = reinterpret_cast<uint32_t *>(sm + KW_SLAB_BYTES);
    uint32_t *cnt = reinterpret_cast<uint32_t *>(sm + KW_SLAB_BYTES + 2048);   // [64] bin totals
    unsigned long long *mbar = reinterpret_cast<unsigned long long *>(sm + KW_SLAB_BYTES + 2048 + 256);

    const int lane = threadIdx.x;
    const uint32_t lt_mask = (1u << lane) - 1u;
    const int mesh = blockIdx.x;
    const int frame = mesh / (a.ny * a.nx);
    const int mj = (mesh / a.nx) % a.ny, mi = mesh % a.nx;
    const int y0 = mj * a.mh, x0 = mi * a.mw;
    const int vh = min(a.mh, a.H - y0), vw = min(a.mw, a.W - x0);
    const int n_tot = vh * vw, n4 = n_tot >> 2;
    const float *mesh_ptr = a.img + (size_t)frame * a.H * a.W + (size_t)y0 * a.W + x0;

    int reason = 0;
    if (n_tot < KW_MIN_PX || vw < 16) reason = 7;
    double med = 0, mu = 0, sd = 0;
    int n_final = n_tot;

    if (!reason) {
        // ---- stage the mesh: one TMA bulk-tensor load (full-width meshes), else a plain packed copy ------------------
        if (a.use_tma && vw == a.mw) {
            const uint32_t bar = smem_u32(mbar);
            if (lane == 0) {
                asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar));
                asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
                asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"((uint32_t)(a.mh * a.mw * 4)) : "memory");
                // rows past H are zero-filled; they lie beyond the n_tot prefix and are never read
                asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
                             ::"r"(slab_s), "l"(&tmap), "r"(x0), "r"(y0), "r"(frame), "r"(bar) : "memory");
            }
            __syncwarp();
            uint32_t done = 0;
            while (!done)
                asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0; selp.u32 %0, 1, 0, p; }"
                             : "=r"(done) : "r"(bar) : "memory");
        } else {
            const int f4_row = vw >> 2;
            for (int i = lane; i < n4; i += 32) {
                const int r = i / f4_row, c = i - r * f4_row;
                const float4 v = __ldg(reinterpret_cast<const float4 *>(mesh_ptr + (size_t)r * a.W) + c);
                reinterpret_cast<float4 *>(sm)[i] = v;
            }
            __syncwarp();
        }

        // ---- lattice sample (8 x 8 points x 4 consecutive pixels), sorted in registers --------------------------------
        uint32_t x[8];
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            const int e = r * 32 + lane, pt = e >> 2, q = e & 3, i = pt >> 3, j = pt & 7;
            const int y = ((2 * i + 1) * vh) >> 4;
            const int xx = min((((2 * j + 1) * vw) >> 4) & ~3, vw - 4) + q;
            x[r] = kw_lds32(slab_s + 4u * (uint32_t)(y * vw + xx));   // raw float bits
        }
#pragma unroll
        for (int r = 0; r < 8; ++r) x[r] = f32_to_key(__uint_as_float(x[r]));
        kw_sort256(x, lane);
        // sorted rank rho sits in lane rho / 8, register rho % 8
        const double q50 = (double)key_to_f32(__shfl_sync(0xffffffffu, x[0], 128 / 8));
        const double q16 = (double)key_to_f32(__shfl_sync(0xffffffffu, x[0], 40 / 8));
        const uint32_t ka = __shfl_sync(0xffffffffu, x[0], 88 / 8);     // +-5 standard deviations of a 256-sample median
        const uint32_t kb = __shfl_sync(0xffffffffu, x[0], 168 / 8);
        const double sig = q50 - q16;    // lower side: sources and hot pixels are positive
        const double pivot = q50;
        const float A_f = (float)(pivot - 2.0 * sig), B_f = (float)(pivot + 2.0 * sig);
        if (!(sig > 0.0) || ka >= kb || !((double)A_f < pivot) || !((double)B_f > pivot)) reason = 1;

        if (!reason) {
            // ---- the sweep: core sums, count below the bracket, in-place list L of tail pixels and bracket candidates ---
            const uint32_t span = kb - ka;
            const int shift = max(0, 26 - __clz(span));   // smallest shift with (span >> shift) < 64
            double t1 = 0.0, t2 = 0.0;
            int c_core = 0;
            uint32_t below = 0, m = 0;
            for (int i0 = 0; i0 < n4; i0 += 32) {
                const bool ok = i0 + lane < n4;
                uint4 v = make_uint4(0, 0, 0, 0);
                if (ok) v = kw_lds128(slab_s + 16u * (uint32_t)(i0 + lane));
                // L grows over slab words that OTHER lanes load in this same iteration (m <= 4 i0): every lane's load must
                // have completed before the first store below.  The vote intrinsics order nothing in memory; this does.
                __syncwarp();
                const uint32_t raw[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const float e = __uint_as_float(raw[q]);
                    const uint32_t k = f32_to_key(e);
                    const bool incore = ok && e >= A_f && e <= B_f;
                    if (incore) {
                        const double d = (double)e - pivot;
                        t1 += d;
                        t2 = fma(d, d, t2);
                        ++c_core;
                    }
                    below += (ok && k < ka) ? 1u : 0u;
                    const bool keep = ok && (!incore || (k - ka) <= span);
                    const uint32_t bal = __ballot_sync(0xffffffffu, keep);
                    if (keep) kw_sts32(slab_s + 4u * (m + __popc(bal & lt_mask)), k);
                    m += __popc(bal);
                }
            }
            t1 = kw_sum(t1); t2 = kw_sum(t2);
            const int n_core = kw_sum(c_core);
            const uint32_t off = (uint32_t)kw_sum((int)below);
            __syncwarp();

            // ---- 64-bin histogram of the candidates (per-lane byte columns: a lane sees <= 128 entries) -----------------
#pragma unroll
            for (int k = 0; k < 4; ++k) reinterpret_cast<uint4 *>(hist8)[k * 32 + lane] = make_uint4(0, 0, 0, 0);
            __syncwarp();
            for (uint32_t j0 = 0; j0 < m; j0 += 32) {
                const uint32_t j = j0 + lane;
                if (j < m) {
                    const uint32_t t = kw_lds32(slab_s + 4u * j) - ka;
                    if (t <= span) hist8[(t >> shift) * 32 + lane] += 1;
                }
            }
            __syncwarp();
            uint32_t c0 = 0, c1 = 0;
            {
                const uint32_t *row = reinterpret_cast<const uint32_t *>(hist8) + 16 * lane;   // bins 2 lane, 2 lane + 1
#pragma unroll
                for (int w = 0; w < 8; ++w) {
                    const int ww = (w + lane) & 7;   // rotated: spreads the lanes over the banks
                    c0 = __dp4a(row[ww], 0x01010101u, c0);
                    c1 = __dp4a(row[8 + ww], 0x01010101u, c1);
                }
            }
            cnt[2 * lane] = c0; cnt[2 * lane + 1] = c1;
            __syncwarp();
            // A window of bins around the bin that holds a wanted rank, with <= KW_WIN keys, gathered from L and sorted in
            // registers; every lane computes the same bins.  Later rounds clip mostly positive outliers, which moves the
            // median rank DOWN: two bins on the low side for every bin on the high side.  Built for the round-0 median;
            // a round whose rank has left it (crowded meshes lose 10 % of their pixels to the clipping) builds it again.
            const int nb = (int)(span >> shift) + 1;
            uint32_t list_off = 0, m_win = 0;
            auto build_window = [&](uint32_t want) -> int {   // want: 0-based rank among the candidates; returns a reason
                int b_hit = -1;
                uint32_t run = 0;
                for (int b = 0; b < nb; ++b) {
                    const uint32_t c = cnt[b];
                    if (want < run + c) { b_hit = b; break; }
                    run += c;
                }
                if (b_hit < 0) return 3;
                if (cnt[b_hit] > (uint32_t)KW_WIN) return 4;
                int b0 = b_hit, b1 = b_hit;
                uint32_t tot = cnt[b_hit], pre0 = run;
                for (int g = 0; g < 64; ++g) {
                    bool grew = false;
                    for (int rep = 0; rep < 2; ++rep)
                        if (b0 - 1 >= 0 && tot + cnt[b0 - 1] <= (uint32_t)KW_WIN) { --b0; tot += cnt[b0]; pre0 -= cnt[b0]; grew = true; }
                    if (b1 + 1 < nb && tot + cnt[b1 + 1] <= (uint32_t)KW_WIN) { ++b1; tot += cnt[b1]; grew = true; }
                    if (!grew) break;
                }
                list_off = off + pre0; m_win = tot;
                const uint32_t kga = ka + ((uint32_t)b0 << shift);
                const uint32_t kgb = min(kb, ka + ((((uint32_t)b1 + 1u) << shift) - 1u));
                const uint32_t gspan = kgb - kga;
                __syncwarp();   // the histogram (first call) / the previous window is dead
                uint32_t mw_ = 0;
                for (uint32_t j0 = 0; j0 < m; j0 += 32) {
                    const uint32_t j = j0 + lane;
                    const uint32_t k = j < m ? kw_lds32(slab_s + 4u * j) : 0u;
                    const bool in = j < m && (k - kga) <= gspan;
                    const uint32_t bal = __ballot_sync(0xffffffffu, in);
                    if (in) win[mw_ + __popc(bal & lt_mask)] = k;
                    mw_ += __popc(bal);
                }
                __syncwarp();
#pragma unroll
                for (int r = 0; r < 8; ++r) x[r] = (uint32_t)(lane * 8 + r) < m_win ? win[lane * 8 + r] : 0xFFFFFFFFu;
                kw_sort256(x, lane);
                __syncwarp();
#pragma unroll
                for (int r = 0; r < 8; ++r) win[lane * 8 + r] = x[r];
                __syncwarp();
                return 0;
            };
            const uint32_t k_first = (uint32_t)((n_tot - 1) / 2);
            // the tail list T goes behind L (L stays: the window may be rebuilt), so both must fit the slab
            uint32_t mt = 0;
            if (!(n_core > 0 && k_first >= off)) reason = 3;
            else {
                uint32_t n_tail_px = (uint32_t)(n_tot - n_core);
                if (m + n_tail_px > (uint32_t)(KW_SLAB_BYTES / 4)) reason = 2;
            }
            if (!reason) reason = build_window(k_first - off);
            if (!reason) {
                // ---- tail entries of L, copied behind it ------------------------------------------------------------------
                const uint32_t T_s = slab_s + 4u * m;
                for (uint32_t j0 = 0; j0 < m; j0 += 32) {
                    const uint32_t j = j0 + lane;
                    const uint32_t k = j < m ? kw_lds32(slab_s + 4u * j) : 0u;
                    const float e = key_to_f32(k);
                    const bool tl = j < m && !(e >= A_f && e <= B_f);
                    const uint32_t bal = __ballot_sync(0xffffffffu, tl);
                    if (tl) kw_sts32(T_s + 4u * (mt + __popc(bal & lt_mask)), k);
                    mt += __popc(bal);
                }
                __syncwarp();
                // ---- clipping rounds on the tail list (readings A5-A7) ----------------------------------------
                const double A_d = (double)A_f, B_d = (double)B_f;
                auto tail_stats = [&](double lo, double hi, double &q1, double &q2, int &c_in, int &c_below) {
                    q1 = 0; q2 = 0; c_in = 0; c_below = 0;
                    for (uint32_t j = lane; j < mt; j += 32) {
                        const double xv = (double)key_to_f32(kw_lds32(T_s + 4u * j));
                        if (xv < lo) ++c_below;
                        else if (xv <= hi) {
                            const double d = xv - pivot;
                            ++c_in;
                            q1 += d;
                            q2 = fma(d, d, q2);
                        }
                    }
                    q1 = kw_sum(q1); q2 = kw_sum(q2); c_in = kw_sum(c_in); c_below = kw_sum(c_below);
                };
                double LO = -INFINITY, HI = INFINITY, q1, q2;
                int c_in, c_below;
                tail_stats(LO, HI, q1, q2, c_in, c_below);
                int n = n_core + c_in, n_below = c_below;
                double s1 = t1 + q1, s2 = t2 + q2;
                for (int round = 0;; ++round) {
                    const double inv_n = 1.0 / (double)n;
                    const double m1 = s1 * inv_n;
                    mu = pivot + m1;
                    const double var = s2 * inv_n - m1 * m1;
                    sd = var > 0.0 ? sqrt(var) : 0.0;
                    const uint32_t k0 = (uint32_t)(n_below + (n - 1) / 2);
                    const bool two = (n & 1) == 0;
                    if (k0 < list_off || k0 + (two ? 1u : 0u) >= list_off + m_win) {   // the rank left the window: build it again
                        if (k0 < off) { reason = 5; break; }
                        reason = build_window(k0 - off);
                        if (!reason && (k0 < list_off || k0 + (two ? 1u : 0u) >= list_off + m_win)) reason = 5;
                        if (reason) break;
                    }
                    const uint32_t jj = k0 - list_off;
                    const uint32_t key_a = win[jj], key_b = two ? win[jj + 1] : key_a;
                    med = 0.5 * ((double)key_to_f32(key_a) + (double)key_to_f32(key_b));
                    n_final = n;
                    if (round >= a.iters) break;
                    const double lo = fmax(LO, med - a.k_c * sd), hi = fmin(HI, med + a.k_c * sd);
                    if (!(lo <= A_d && hi >= B_d)) { reason = 6; break; }   // a bound entered the core
                    tail_stats(lo, hi, q1, q2, c_in, c_below);
                    const int n_new = n_core + c_in;
                    if (n_new == n) break;   // stable (A7); n_new > 0 because the core survives
                    LO = lo; HI = hi;
                    n = n_new; n_below = c_below; s1 = t1 + q1; s2 = t2 + q2;
                }
            }
        }
    }

    if (lane == 0) {
        if (reason) {   // the general kernel takes this mesh
            a.fb_list[atomicAdd(a.fb_count, 1u)] = (uint32_t)mesh;
            if (reason < 7) atomicAdd(&g_k1_reason[reason], 1ull);
        } else {
            double bkg = a.median_factor * med - a.mean_factor * mu;
            if (a.skew_guard) {
                if (sd == 0.0) bkg = mu;
                else if (fabs(mu - med) / sd >= 0.3) bkg = med;
            }
            if (a.bkg_raw) a.bkg_raw[mesh] = bkg;
            if (a.rms_raw) a.rms_raw[mesh] = sd;
            if (a.median) a.median[mesh] = med;
            if (a.mean) a.mean[mesh] = mu;
            if (a.n_kept) a.n_kept[mesh] = n_final;
        }
    }
}
