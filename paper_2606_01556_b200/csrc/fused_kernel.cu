// fused_kernel.cu -- launch planning and dispatch for the fused dual-branch kernel
// (kernel template: fused_kernel.cuh; instantiations: fused_inst_*.cu).  Host arithmetic only.
#include "fused_kernel.cuh"

namespace twq {

namespace {

int pick_tn(int M) { return M <= 16 ? 16 : (M <= 32 ? 32 : (M <= 64 ? 64 : 128)); }

int round_up(int x, int a) { return (x + a - 1) / a * a; }

// Clusters of `cs` CTAs (one CTA per SM) that can be resident at once.  A cluster must sit inside
// one GPC, so this is less than num_sms / cs for large clusters; asked of the driver once per size,
// with a conservative table when no device is present (planning on a CPU-only box).
int cluster_capacity(int cs, int num_sms) {
    if (cs <= 1) return num_sms;
    constexpr int kMaxDevices = 64;
    static int cache[kMaxDevices][9] = {};                 // per device; idempotent values
    int dev = 0;
    const bool have_dev = cudaGetDevice(&dev) == cudaSuccess && dev >= 0 && dev < kMaxDevices - 1;
    if (!have_dev) { cudaGetLastError(); dev = kMaxDevices - 1; }
    if (cache[dev][cs] > 0) return cache[dev][cs];
    int n = have_dev ? max_active_clusters_inst<128, 128, false>(cs, num_sms) : 0;
    if (n <= 0) n = cs == 2 ? num_sms / 2 : (cs == 4 ? (num_sms / 4) * 7 / 8 : (num_sms / 8) * 7 / 8);
    if (n > num_sms / cs) n = num_sms / cs;
    if (n < 1) n = 1;
    cache[dev][cs] = n;
    return n;
}

}  // namespace

// Launch plan: tile size, cluster size, K splits, persistent clusters, ring depths, shared-memory map.
static bool make_plan_tn(int TN, int M, int N, int K, int r, int G, int num_sms, FusedPlan* out) {
    FusedPlan pl = {};
    const int ng = K / G;
    pl.TN = TN;
    pl.n_tiles = (N + kTileN - 1) / kTileN;
    pl.m_tiles = (M + TN - 1) / TN;
    // cluster (shares H when there is a low-rank branch): among 8/4/2/1 dividing the n-tiles, the size
    // that keeps the most SMs busy; ties go to the larger cluster (less redundant stage-1 work)
    pl.cs = 1;
    if (r > 0) {
        const long long tiles0 = static_cast<long long>(pl.n_tiles) * pl.m_tiles;
        // (a K split needs room for at least two splits per tile; between num_sms / 2 and 3/4 num_sms tiles the call runs unsplit
        // on fewer SMs, and the cost model below picks the cluster: Qwen3 attention, 80 tiles at M = 128: 46.1 us with clusters
        // of 2, 40.7 / 41.9 us with 4 / 8)
        if (tiles0 < (3 * num_sms) / 4 && 2 * tiles0 <= num_sms) {
            // few tiles (K will be split): the size that keeps the most SMs busy; ties go to the larger cluster
            int best = 0;
            for (int c = 8; c >= 1; c >>= 1) {
                if (pl.n_tiles % c != 0) continue;
                const int sms = cluster_capacity(c, num_sms) * c;
                if (sms > best + best / 16) { best = sms; pl.cs = c; }
            }
        } else {
            // unsplit path: a cost model in cycles per CTA.  A cluster recomputes H = X*L1 once per token tile it
            // touches, each CTA a serial chain of K/(64*cs) chunks (~700 cycles each); the residual costs ~1450 cycles
            // per K-group per tile (both fitted to gate/up and down at M = 2048 over cs = 2 / 4 / 8, r01c).  Small
            // clusters cover more SMs, large ones share stage 1 further.
            long long best_cost = -1;
            for (int c = 8; c >= 1; c >>= 1) {
                if (pl.n_tiles % c != 0) continue;
                const int nb = pl.n_tiles / c;
                const long long units = static_cast<long long>(pl.m_tiles) * nb;
                const long long ncl = units < cluster_capacity(c, num_sms) ? units : cluster_capacity(c, num_sms);
                const long long upc = (units + ncl - 1) / ncl;                       // units per cluster (the longest)
                const long long ctxs = (upc + nb - 1) / nb + ((upc > 1 && nb > 1) ? 1 : 0);
                const long long cost = ctxs * ((K / 64 + c - 1) / c) * 700 + upc * ng * 1450;
                if (best_cost < 0 || cost < best_cost) { best_cost = cost; pl.cs = c; }
            }
        }
    }
    const unsigned flags = plan_flags();                  // test overrides (include/twq_testing.h); 0 in production
    {
        const int c = static_cast<int>((flags >> kPlanFusedCsShift) & 15u);
        if (r > 0 && (c == 1 || c == 2 || c == 4 || c == 8) && pl.n_tiles % c == 0) pl.cs = c;
    }
    pl.n_blocks = pl.n_tiles / pl.cs;
    const int max_clusters = cluster_capacity(pl.cs, num_sms);
    // K splits when the output tiles alone cannot fill the machine (decode-shaped M)
    const long long tiles = static_cast<long long>(pl.n_tiles) * pl.m_tiles;
    int s = 1;
    // kPlanNoSplit: testing aid -- small shapes then take the unsplit path (and CTA pairs) of large ones
    if (tiles < (3 * num_sms) / 4 && !(flags & kPlanNoSplit)) {
        s = static_cast<int>(static_cast<long long>(max_clusters) * pl.cs / tiles);
        if (s > 16) s = 16;
        if (s > ng) s = ng;
        if (s < 1) s = 1;
    }
    pl.g_per_split = (ng + s - 1) / s;
    pl.splits = (ng + pl.g_per_split - 1) / pl.g_per_split;   // every split non-empty
    pl.units = pl.splits * pl.m_tiles * pl.n_blocks;
    pl.nclusters = pl.units < max_clusters ? pl.units : max_clusters;
    if (pl.splits > 1 && pl.nclusters != pl.units) {          // the fix-up assumes one unit per cluster
        pl.splits = 1;
        pl.g_per_split = ng;
        pl.units = pl.m_tiles * pl.n_blocks;
        pl.nclusters = pl.units < max_clusters ? pl.units : max_clusters;
    }
    // shared memory map
    const int nrb = (r + 127) / 128, nkb = (r + 63) / 64;
    const int hbytes = nkb * TN * 128, l2bytes = nkb * kL1Chunk;
    // CTA pairs: prefill tiles in an even cluster without K splits; each CTA then expands half of the token rows
    pl.pair = (TN == 128 && pl.cs >= 2 && pl.splits == 1 && !(flags & kPlanNoPair)) ? 1 : 0;
    const int xr = pl.pair ? TN / 2 : TN;
    const int ub = xr * G, pb = kTileN * (G / 2) + xr * (G / 2);
    const int s1b = TN * 128 + nrb * kL1Chunk;
    const int hpart = pl.cs > 1 ? round_up(TN * r * 4, 1024) : 0;
    const int fixed = kSxSlots * TN * 4 + B_COUNT * 8 + 256;
    const int budget = kMaxDynSmem - 1024 - fixed;             // dynamic limit minus alignment slack
    // output staging for the asynchronous (TMA) store of a finished 128-token tile of 16-bit outputs: two 128-byte-
    // swizzled halves of 64 channels; taken only where it fits beside a packed ring of at least 6 (pairs) / 4 stages.
    // The caller clears the flag for FP32 outputs and row pitches that are not a multiple of 16 bytes.
    const int ybytes = TN * kTileN * 2;
    pl.ystage = (TN == 128 && pl.splits == 1 && !(flags & kPlanNoYStage)) ? 1 : 0;
    pl.nsu = kMaxNSU;
    pl.nsp = pl.pair ? kMaxNSP : (TN <= 32 ? 5 : (TN == 64 ? 3 : 4));   // a pair's packed stage is 12 KB: the ring can be twice as deep
    pl.ns1 = r > 0 ? (TN <= 32 ? 3 : 2) : 0;
    pl.alias = 0;
    auto total = [&](const FusedPlan& q) {
        const int resid = q.nsu * ub + round_up(q.nsp * pb, 1024);
        const int s1 = q.alias ? (q.ns1 * s1b > hpart ? q.ns1 * s1b : hpart) : q.ns1 * s1b + hpart;
        const int ys = q.ystage ? ybytes + 1024 : 0;
        if (q.alias == 2) return hbytes + (l2bytes + resid > s1 ? l2bytes + resid : s1) + ys;
        return hbytes + l2bytes + (q.alias ? (resid > s1 ? resid : s1) : resid + s1) + ys;
    };
    if (pl.ystage) {
        FusedPlan q = pl;
        q.alias = 1; q.ns1 = r > 0 ? 3 : 0;
        if (total(q) > budget && pl.pair) q.nsp = 6;
        if (total(q) > budget) pl.ystage = 0;
        else if (total(pl) > budget) pl.nsp = q.nsp;
    }
    if (total(pl) > budget) { pl.alias = 1; pl.ns1 = r > 0 ? 3 : 0; }
    // split-K calls run ONE unit per cluster, so the overlay of the stage-1 ring on the residual rings never makes a
    // tile wait for its predecessor: take it, and with it the deepest stage-1 ring
    if (pl.splits > 1 && r > 0 && pl.alias == 0) { pl.alias = 1; pl.ns1 = kMaxNS1; }
    if (total(pl) > budget && r > 0 && !(flags & kPlanNoAlias2)) {
        // Rank-256 buffers beside a 128-token tile: the stage-1 ring and the FP32 partial of H overlay the L2T tile as
        // well as the residual rings.  L2T is dead whenever stage 1 runs: its stage-2 MMAs were issued at the start
        // of the previous tile, whose residual MMAs (B_RESID) the producer waits for before the first stage-1 load,
        // and the next L2T load follows B_HREADY (the same two waits that protect the rings).
        FusedPlan q = pl;
        q.alias = 2;
        q.ystage = 0;
        while (total(q) > budget && q.nsp > 4) --q.nsp;
        if (total(q) <= budget) pl = q;
    }
    // a deeper stage-1 ring wherever it costs nothing (it overlays the residual rings) or still fits: every chunk of the
    // stage-1 chain is a round trip to L2 / HBM, and with two stages in flight the chain ran at one round trip per chunk
    // (in-kernel timeline at M = 128, r02: 2600 cycles per 64-wide chunk, 11 of the call's 29 us)
    while (r > 0 && pl.ns1 < kMaxNS1) {
        FusedPlan q = pl;
        ++q.ns1;
        if (total(q) > budget) break;
        pl = q;
    }
    while (total(pl) > budget && pl.nsp > 2) --pl.nsp;
    while (total(pl) > budget && pl.nsu > 2) --pl.nsu;
    while (total(pl) > budget && pl.ns1 > 2) --pl.ns1;
    if (total(pl) > budget) return false;
    int o = 0;
    pl.off_H = o; o += hbytes;
    pl.off_L2T = o; o += l2bytes;
    pl.off_U = o;
    pl.off_P = o + pl.nsu * ub;
    const int resid = pl.nsu * ub + round_up(pl.nsp * pb, 1024);
    if (pl.alias == 2) {
        pl.off_S1 = pl.off_L2T;
        pl.off_Hpart = pl.off_L2T;
        const int s1 = pl.ns1 * s1b > hpart ? pl.ns1 * s1b : hpart;
        o = pl.off_L2T + (l2bytes + resid > s1 ? l2bytes + resid : s1);
    } else if (pl.alias) {
        pl.off_S1 = o;
        pl.off_Hpart = o;   // the FP32 partial is written after the stage-1 MMAs completed
        const int s1 = pl.ns1 * s1b > hpart ? pl.ns1 * s1b : hpart;
        o += resid > s1 ? resid : s1;
    } else {
        o += resid;
        pl.off_S1 = o; o += pl.ns1 * s1b;
        pl.off_Hpart = o; o += hpart;
    }
    o = round_up(o, 16);
    if (pl.ystage) { o = round_up(o, 1024); pl.off_Y = o; o += ybytes; }
    pl.off_sx = o; o += kSxSlots * TN * 4;
    pl.off_bar = o; o += B_COUNT * 8 + 256;
    pl.smem_bytes = o + 1024;
    pl.tmem_cols = Cfg<16, 128>::kTmemCols;   // informational
    *out = pl;
    return true;
}

bool fused_make_plan(int M, int N, int K, int r, int G, int num_sms, FusedPlan* out) {
    // a smaller token tile is the fallback when rank-256 buffers do not fit beside a 128-token tile
    int tn0 = pick_tn(M);
    const unsigned cap = (plan_flags() >> kPlanFusedTnShift) & 3u;       // test / measurement override
    if (cap == 1 && tn0 > 64) tn0 = 64;
    if (cap == 2 && tn0 > 32) tn0 = 32;
    // Mid-size M: where 128-token tiles alone cannot fill the machine (the plan would split K: partial tiles through L2 and a
    // fix-up pass that move as many bytes as the weights), a smaller token tile WITHOUT a K split wins as soon as it yields
    // enough tiles -- measured on q_proj (4096 x 4096, r = 128): M = 128 as 4 x 32 tokens 24.1 vs 27.5 us, M = 192 as 6 x 32
    // 32.6 vs 36.0, M = 256 as 4 x 64 33.9 vs 36.3; with only 96 tiles (M = 96 as 3 x 32, M = 192 as 3 x 64) it loses.  The largest
    // tile that reaches 85 % of the SMs is taken; no workspace is needed then.  Only for short K and rank <= 128: an unsplit CTA
    // walks all K-groups in series, and on longer layers the K split wins again (down, K = 14336: M = 128 / 256 62.6 / 91.5 us
    // unsplit against 47.3 / 75.5 us split; Qwen3 attention, K = 5120, r = 256, M = 128: 53.5 against 46.1 us).
    if (tn0 == 128 && cap == 0 && !(plan_flags() & kPlanNoSplit) && K / G <= 32 && r <= 128) {
        const long long n_tiles = (N + kTileN - 1) / kTileN;
        if (((M + 127) / 128) * n_tiles < (3 * num_sms) / 4) {
            for (int TN = 64; TN >= 32; TN >>= 1) {
                const long long tiles = ((M + TN - 1) / TN) * n_tiles;
                if (tiles * 100 < static_cast<long long>(num_sms) * 85) continue;
                FusedPlan q;
                if (make_plan_tn(TN, M, N, K, r, G, num_sms, &q) && q.splits == 1) { *out = q; return true; }
                break;
            }
        }
    }
    for (int TN = tn0; TN >= 16; TN >>= 1)
        if (make_plan_tn(TN, M, N, K, r, G, num_sms, out)) return true;
    return false;
}

cudaError_t launch_fused(const FusedMaps& maps, const FusedParams& p, int G, cudaStream_t stream) {
    const bool dbg = p.dbgP != nullptr;
#define TWQ_CASE(tn, g)                                                               \
    if (p.plan.TN == tn && G == g && !p.plan.pair)                                    \
        return dbg ? launch_fused_inst<tn, g, true>(maps, p, stream) : launch_fused_inst<tn, g, false>(maps, p, stream);
    if (p.plan.pair && p.plan.TN == 128 && G == 128)
        return dbg ? launch_fused_inst<128, 128, true, true>(maps, p, stream) : launch_fused_inst<128, 128, false, true>(maps, p, stream);
    if (p.plan.pair && p.plan.TN == 128 && G == 64)
        return dbg ? launch_fused_inst<128, 64, true, true>(maps, p, stream) : launch_fused_inst<128, 64, false, true>(maps, p, stream);
    TWQ_CASE(16, 128) TWQ_CASE(32, 128) TWQ_CASE(64, 128) TWQ_CASE(128, 128)
    TWQ_CASE(16, 64) TWQ_CASE(32, 64) TWQ_CASE(64, 64) TWQ_CASE(128, 64)
#undef TWQ_CASE
    return cudaErrorInvalidValue;
}

}  // namespace twq
