// xengine_pair.cuh -- the X-engine HERK on CTA PAIRS (tcgen05 cta_group::2).  Same mathematics and same direct feed
// as xengine_tc.cuh
// (Sec. 2 Eq. 2; lower station triangle incl. autocorrelations PAPER.md:79, 144).
//
// Why (profiles/r1a_cfg4_ncu_1cta_kernel.md): with 128 x 256 tiles per CTA every time sample costs
// 128 + 256 operand bytes from L2 per 32768 MACs, and at config 4 that is 15 GB of L2 -> SM traffic per
// call = the L2 slice throughput cap; the tensor pipe idles 60 % of the time.  A CTA pair computes a
// 256 x 256 tile of G with one M = 256 instruction: each CTA holds 128 rows of A and only HALF of B's
// columns (the hardware feeds both halves to both tensor cores), so a sample costs 128 + 128 bytes per CTA
// for the same 32768 MACs (and half the shared-memory operand reads).  (A 4-CTA cluster of two pairs with a
// multicast load of the operand their tiles share was built and measured in round 1: 12 % slower at config 4 --
// the multicast saves L2 reads, not bytes delivered to each SM, and couples the two pipelines -- and removed.)
//
// Roles per CTA (320 threads, one CTA per SM, persistent; the tiles come from the dynamic TileFeed below):
//   warp 0      TMA producer (one elected lane of the converged warp): its 128 A rows and its 128 B columns of every pipeline stage; completion
//               bytes of both CTAs are counted on the pair LEADER's `full` barrier
//   warp 1      TMEM allocator (both CTAs) + tcgen05.mma.cta_group::2 issuer (one elected lane of the leader CTA's warp);
//               tcgen05.commit multicasts the `empty` and `tmem full` arrivals to both CTAs;
//               in cluster rank 1 (no MMAs to issue) the same lane is the tile-feed writer
//   warps 2..9  epilogue of this CTA's 128 TMEM lanes (drain_accumulator in xengine_tc.cuh); they release the
//               accumulator by arriving on the leader's `tmem empty` barrier through shared::cluster
#pragma once
#include "xengine_tc.cuh"

namespace xtc {

constexpr int kPairRows = 256;                 // G rows per pair tile
constexpr int kPairBoxes = 1;                  // TMA boxes stacked along time per 128-byte chunk of a pipeline stage
// Six stages of 32 KB: one 16 KB TMA box per operand chunk and 4 MMAs per stage.  History: round 1 had 6 x 32 KB; while the
// MMAs were issued from a divergent `if (lane == 0)` (an elect / R2UR loop of ~90 clk around every instruction) four MMAs
// plus the stage's barrier traffic did not fit into the 512 clk they execute in, and three stages of 64 KB (8 MMAs) were
// 8 - 15 % fewer cycles.  With the issue in uniform control flow (ptx::elect_one) that cost is gone and the finer ring wins:
// 160 instead of 128 KB of operands in flight per CTA while a stage is consumed (the load latency of ~2000 clk is the
// ring's whole period), measured +5 % cross-only, +3 % N = 128, +2 - 4 % fp16, +1 % config 4 / N = 1024.  (12 x 16 KB: -10 %.)
constexpr int kPairStageBytes = 32 * 1024;     // per CTA and stage: A 128 components + B 128 components, kPairStageK samples
template <int kElt> constexpr int kPairStageK = kPairStageBytes / (2 * 128 * kElt);    // 128 (ci8) / 64 (cf16) samples
constexpr int kPairEpiBufs = 1;                // staging buffers per epilogue warp (a second one costs two pipeline stages)
constexpr int kPairEpiWarpBytes = kPairEpiBufs * kEpiBufBytes;
constexpr int kPairEpiBytes = kNumEpiWarps * kPairEpiWarpBytes;
constexpr int kPairStages = 6;
// the dynamic shared memory window of a kernel without static shared memory starts 1024-byte aligned (checked
// in the kernel), so no alignment slack is reserved
constexpr int kPairSmemBytes = kPairStages * kPairStageBytes + kPairEpiBytes + 256 /*barriers*/;
static_assert(kPairSmemBytes <= 227 * 1024, "shared memory");

struct PairTile {
    int row0;   // first G row    (multiple of 256), real components u within the channel
    int col0;   // first G column (multiple of 256)
};

struct PairParams {
    Params base;                 // geometry, output, accumulate, k_chunk (tiles/tiles_per_chan/n_tiles unused)
    const PairTile* tiles;       // DEVICE: per-channel tile table (triangle: column-block major; rectangle: all blocks)
    int tiles_per_chan;
    long long n_tiles;           // tiles_per_chan * n_chan * n_dump (< 2^31 - grid)
    unsigned int* sched_counter; // DEVICE, zeroed before the launch: tiles handed out beyond the first one per cluster
};

// Dynamic tile feed.  Every cluster starts on tile `cluster id`; further tiles are claimed in order from one
// global counter, so all clusters work on neighbouring tiles (= the same few channels: their input stays in L2) and a
// slow cluster simply takes fewer tiles (a static round robin ended 9.5 % later on its slowest cluster).  The
// otherwise idle MMA-warp lane of cluster rank 1 (the pair's second CTA issues no MMAs) is the writer: it claims tiles
// with atomicAdd and publishes each into a small slot ring in the shared memory of BOTH CTAs
// (st.shared::cluster + cluster-scope fence + remote mbarrier arrive); producers, the MMA issuer and epilogue warps read
// their CTA's copy and report the slot read on rank 1's `slot free` barrier.  A value >= n_tiles ends every loop.
// (Claiming from the TMA producer thread instead cost 1500 clk per tile of load issue: measured 13 % slower.)
constexpr int kFeedSlots = 3;      // the writer claims at most this many tiles ahead of the cluster's slowest reader
struct TileFeed {
    uint32_t full0;           // this CTA's  slot-filled barriers  [kFeedSlots]
    uint32_t slot0;           // this CTA's  slot values (u32)     [kFeedSlots]
    uint32_t free0_writer;    // rank 1's    slot-free barriers    [kFeedSlots], shared::cluster address
    int slot;
    uint32_t phase;
    __device__ __forceinline__ TileFeed(uint32_t full0_, uint32_t free0_, uint32_t slot0_)
        : full0(full0_), slot0(slot0_), free0_writer(ptx::mapa(free0_, 1)), slot(0), phase(0) {}
    __device__ __forceinline__ void advance() {
        if (++slot == kFeedSlots) { slot = 0; phase ^= 1u; }
    }
    // one consumer thread
    __device__ __forceinline__ long long next() {
        ptx::mbar_wait_cluster(full0 + 8u * slot, phase);
        const uint32_t g = ptx::ld_shared_u32(slot0 + 4u * slot);
        ptx::mbar_arrive_cluster_after(free0_writer + 8u * slot, g);
        advance();
        return g;
    }
    // a whole (converged) warp: every lane reads, lane 0 reports (vote-based wait: the lanes leave the poll together, so the
    // __syncwarp below and the .sync.aligned tcgen05.ld that follow find the warp converged; see ptx::mbar_wait_uniform)
    __device__ __forceinline__ long long next_warp(int lane) {
        ptx::mbar_wait_cluster_uniform(full0 + 8u * slot, phase);
        const uint32_t g = ptx::ld_shared_u32(slot0 + 4u * slot);
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive_cluster_after(free0_writer + 8u * slot, g);
        advance();
        return g;
    }
    // a whole (converged) warp whose control flow must stay provably warp-uniform (TMA producer, MMA issuer)
    __device__ __forceinline__ long long next_uniform(int lane) {
        ptx::mbar_wait_cluster_uniform(full0 + 8u * slot, phase);
        const uint32_t g = ptx::ld_shared_u32(slot0 + 4u * slot);
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive_cluster_after(free0_writer + 8u * slot, g);
        advance();
        return ptx::uniform(g);
    }
    // the writer (one thread of cluster rank 1; `free0_local` is its own barrier): same slot/phase bookkeeping
    __device__ __forceinline__ void publish(uint32_t g, uint32_t free0_local) {
        ptx::mbar_wait(free0_local + 8u * slot, phase ^ 1u);         // every consumer of the cluster has read the old value
        for (uint32_t r = 0; r < 2; ++r) ptx::st_shared_cluster_u32(ptx::mapa(slot0 + 4u * slot, r), g);
        ptx::fence_acq_rel_cluster();
        for (uint32_t r = 0; r < 2; ++r) ptx::mbar_arrive_cluster(ptx::mapa(full0 + 8u * slot, r));
        advance();
    }
};

template <int kElt>
__global__ void __launch_bounds__(kNumThreads, 1)
xengine_pair_kernel(const __grid_constant__ CUtensorMap tmap_in, const __grid_constant__ CUtensorMap tmap_b,
                    const PairParams pp) {
    using C = Cfg<kElt>;
    const Params& prm = pp.base;
    constexpr int kChunkElems = 128 / kElt;                 // u per 128-byte chunk
    constexpr int kStageK = kPairStageK<kElt>;              // samples per pipeline stage
    constexpr int kBoxRows = kStageK / kPairBoxes;          // one TMA box: [kBoxRows samples][128 B] (tmap_pair)
    constexpr int kBoxBytes = kBoxRows * 128;
    constexpr int kChunkBytes = kStageK * 128;              // one 128-byte-wide chunk of a stage (boxes stacked along K)
    constexpr int kOpChunks = 128 / kChunkElems;            // chunks per operand and CTA: 1 (ci8) / 2 (cf16)
    constexpr int kKStepBytes = C::kMmaK * 128;
    constexpr int kKSteps = kStageK / C::kMmaK;
    static_assert(2 * kOpChunks * kChunkBytes == kPairStageBytes, "stage size");
    // M = 256 (16 << 24), N = 256 (32 << 17); formats and MN-major bits as for the 1-CTA kernel
    constexpr uint32_t kIdesc = (C::kIdesc & ~(0x1fu << 24)) | (16u << 24) | (32u << 17);
    constexpr uint16_t kPairMask = 3;

    extern __shared__ uint8_t smem_raw[];
    // the SAME offsets in both CTAs of the pair (cta_group::2 addresses by offset): the dynamic shared memory
    // window starts at the same offset in all CTAs of a launch.  SWIZZLE_128B needs 1024-byte alignment; a kernel
    // without static shared memory gets it (corr_create verifies the launch works; a violation traps).
    const uint32_t smem_base = ptx::smem_u32(smem_raw);
    if (smem_base & 1023u) __trap();
    const uint32_t epi_base = smem_base + kPairStages * kPairStageBytes;
    const uint32_t bar_base = epi_base + kPairEpiBytes;
    auto full_bar = [&](int s) { return bar_base + 8u * s; };
    auto empty_bar = [&](int s) { return bar_base + 8u * (kPairStages + s); };
    auto tfull_bar = [&](int a) { return bar_base + 8u * (2 * kPairStages + a); };
    auto tempty_bar = [&](int a) { return bar_base + 8u * (2 * kPairStages + 2 + a); };
    const uint32_t tmem_slot = bar_base + 8u * (2 * kPairStages + 4);
    const uint32_t feed_full0 = bar_base + 8u * (2 * kPairStages + 5);
    const uint32_t feed_free0 = feed_full0 + 8u * kFeedSlots;
    const uint32_t feed_slot0 = feed_free0 + 8u * kFeedSlots;
    static_assert(8 * (2 * kPairStages + 5 + 2 * kFeedSlots) + 4 * kFeedSlots <= 256, "barrier region");
    // readers of a feed slot per cluster: 8 epilogue warps and the TMA producer of each CTA, and the MMA issuer
    constexpr uint32_t kFeedReaders = 2 * kNumEpiWarps + 2 + 1;
    uint32_t* tmem_slot_ptr = reinterpret_cast<uint32_t*>(smem_raw + (tmem_slot - ptx::smem_u32(smem_raw)));

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;
    // (special registers read through asm: made provably warp-uniform so that the single-thread instruction streams below
    // keep their operands in uniform registers, see ptx::elect_one)
    const int half = static_cast<int>(ptx::uniform(ptx::cluster_ctarank()));      // 0 = pair leader (issues the MMAs)
    const long long cluster_id = ptx::uniform(ptx::cluster_id_x());
    const long long n_clusters = ptx::uniform(ptx::cluster_count_x());

    if (threadIdx.x == 0) {
        ptx::prefetch_tensormap(&tmap_in);
        ptx::prefetch_tensormap(&tmap_b);
        for (int s = 0; s < kPairStages; ++s) {
            ptx::mbar_init(full_bar(s), 1);                  // leader: its own arrive.expect_tx
            ptx::mbar_init(empty_bar(s), 1);                 // the tcgen05.commit arrival
        }
        for (int a = 0; a < 2; ++a) {
            ptx::mbar_init(tfull_bar(a), 1);
            ptx::mbar_init(tempty_bar(a), 2 * kNumEpiWarps); // leader: every epilogue warp of both CTAs
        }
        for (int k = 0; k < kFeedSlots; ++k) {
            ptx::mbar_init(feed_full0 + 8u * k, 1);          // the writer's arrive
            ptx::mbar_init(feed_free0 + 8u * k, kFeedReaders);   // used in rank 1 only
        }
        ptx::fence_mbar_init();
    }
    if (warp == 1) {
        ptx::tmem_alloc_pair(tmem_slot, 512);
        ptx::tmem_relinquish_pair();
    }
    ptx::tc_fence_before();
    ptx::cluster_sync();                 // barriers of both CTAs initialised before anyone signals them
    ptx::tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_ptr;

    const int num_kb = (prm.n_time + kStageK - 1) / kStageK;
    const int kb_per_chunk = prm.k_chunk / kStageK > 0 ? prm.k_chunk / kStageK : 1;
    const int n_kchunks = (num_kb + kb_per_chunk - 1) / kb_per_chunk;
    const int M2 = 2 * prm.M;                                  // G rows per channel (group A in cross mode)
    const bool rect = prm.n_station_b > 0;                     // rectangular cross-only mode: B columns from tmap_b
    const int M2b = rect ? 2 * prm.M_b : M2;                   // G columns per channel

    if (warp == 0) {
        // ===================== TMA producer (whole warp in uniform control flow, one elected lane issues) =====================
        {
            int stage = 0;
            uint32_t phase = 0;
            TileFeed feed(feed_full0, feed_free0, feed_slot0);
            for (long long g = cluster_id; g < pp.n_tiles; g = feed.next_uniform(lane)) {
                const int cd = static_cast<int>(g / pp.tiles_per_chan);             // integration * C + channel
                const PairTile* tdp = pp.tiles + (g - static_cast<long long>(cd) * pp.tiles_per_chan);
                const int row0 = static_cast<int>(ptx::uniform(tdp->row0)), col0 = static_cast<int>(ptx::uniform(tdp->col0));
                const int dump = cd / prm.n_chan, c = prm.chan0 + (cd - dump * prm.n_chan);
                const int w_a = c * M2 + row0 + 128 * half;         // this CTA's A rows in the [n_dump][T][C*2M] view
                const int w_b = c * M2b + col0 + 128 * half;        // this CTA's half of the B columns
                // diagonal tile: this CTA's half of the B columns IS its 128 A rows -> one load serves both operands
                const bool diag = !rect && row0 == col0;
                for (int kb = 0; kb < num_kb; ++kb) {
                    ptx::mbar_wait_uniform(empty_bar(stage), phase ^ 1u);
                    const uint32_t sa = smem_base + stage * kPairStageBytes;
                    const uint32_t sb = sa + kOpChunks * kChunkBytes;
                    if (ptx::elect_one()) {
                        if (half == 0) ptx::mbar_arrive_expect_tx(full_bar(stage), diag ? kPairStageBytes : 2u * kPairStageBytes);
#pragma unroll
                        for (int ch = 0; ch < kOpChunks; ++ch)
#pragma unroll
                            for (int b = 0; b < kPairBoxes; ++b)
                                ptx::tma_load_3d_pair(sa + ch * kChunkBytes + b * kBoxBytes, &tmap_in, full_bar(stage),
                                                      w_a + ch * kChunkElems, kb * kStageK + b * kBoxRows, dump);
                        if (!diag) {
#pragma unroll
                            for (int ch = 0; ch < kOpChunks; ++ch)
#pragma unroll
                                for (int b = 0; b < kPairBoxes; ++b)
                                    ptx::tma_load_3d_pair(sb + ch * kChunkBytes + b * kBoxBytes, &tmap_b, full_bar(stage),
                                                          w_b + ch * kChunkElems, kb * kStageK + b * kBoxRows, dump);
                        }
                    }
                    __syncwarp();
                    if (++stage == kPairStages) { stage = 0; phase ^= 1u; }
                }
            }
        }
    } else if (warp == 1) {
        // ===================== MMA issuer (pair leader only; whole warp in uniform control flow, one elected lane issues) ==
        if (half == 0) {
            const uint32_t tb = ptx::uniform(tmem_base);
            int stage = 0;
            uint32_t phase = 0;
            int acc = 0;
            uint32_t acc_phase = 0;
            TileFeed feed(feed_full0, feed_free0, feed_slot0);
            for (long long g = cluster_id; g < pp.n_tiles; g = feed.next_uniform(lane)) {
                const PairTile* tdp = pp.tiles + g % pp.tiles_per_chan;
                const bool diag = !rect && ptx::uniform(tdp->row0) == ptx::uniform(tdp->col0);      // B operand = the A buffer
                for (int kb0 = 0; kb0 < num_kb; kb0 += kb_per_chunk) {
                    const int kb1 = kb0 + kb_per_chunk < num_kb ? kb0 + kb_per_chunk : num_kb;
                    const uint32_t d_tmem = tb + acc * kTileCols;
                    ptx::mbar_wait_uniform(tempty_bar(acc), acc_phase ^ 1u);     // both CTAs' epilogues have drained it
                    ptx::tc_fence_after();
                    for (int kb = kb0; kb < kb1; ++kb) {
                        ptx::mbar_wait_uniform(full_bar(stage), phase);          // both CTAs' operand bytes have landed
                        ptx::tc_fence_after();
                        const uint32_t sa = smem_base + stage * kPairStageBytes;
                        const uint32_t sb = diag ? sa : sa + kOpChunks * kChunkBytes;
                        if (ptx::elect_one()) {
#pragma unroll
                            for (int k = 0; k < kKSteps; ++k) {
                                const uint64_t adesc = ptx::smem_desc_sw128(sa + k * kKStepBytes, kChunkBytes, 1024);
                                const uint64_t bdesc = ptx::smem_desc_sw128(sb + k * kKStepBytes, kChunkBytes, 1024);
                                const uint32_t accum = (kb != kb0 || k != 0) ? 1u : 0u;
                                if constexpr (C::kFloat) ptx::mma_f16_pair(d_tmem, adesc, bdesc, kIdesc, accum);
                                else ptx::mma_i8_pair(d_tmem, adesc, bdesc, kIdesc, accum);
                            }
                            ptx::mma_commit_pair_mc(empty_bar(stage), kPairMask);  // slot free in both CTAs
                            if (kb + 1 == kb1) ptx::mma_commit_pair_mc(tfull_bar(acc), kPairMask);   // accumulator complete in both CTAs
                        }
                        __syncwarp();
                        if (++stage == kPairStages) { stage = 0; phase ^= 1u; }
                    }
                    if (++acc == 2) { acc = 0; acc_phase ^= 1u; }
                }
            }
        } else if (lane == 0) {
            // ===================== tile-feed writer (this CTA issues no MMAs) =====================
            TileFeed feed(feed_full0, feed_free0, feed_slot0);
            for (;;) {
                const uint32_t g_next = atomicAdd(pp.sched_counter, 1u) + static_cast<uint32_t>(n_clusters);
                feed.publish(g_next, feed_free0);
                if (g_next >= pp.n_tiles) break;
            }
        }
    } else {
        // ===================== epilogue: this CTA's 128 rows of the pair tile =====================
        const int ew = warp - 2;
        const int quarter = warp & 3;                // TMEM lanes [32*quarter, 32*quarter+32) belong to this warp
        const int chalf = ew >> 2;                   // column half of the tile handled by this warp
        const uint32_t stage_smem = epi_base + ew * kPairEpiWarpBytes;
        int acc = 0;
        uint32_t acc_phase = 0;
        int buf = 0;
        TileFeed feed(feed_full0, feed_free0, feed_slot0);
        for (long long g = cluster_id; g < pp.n_tiles; g = feed.next_warp(lane)) {
            const int cd = static_cast<int>(g / pp.tiles_per_chan);
            const PairTile td = pp.tiles[g - static_cast<long long>(cd) * pp.tiles_per_chan];
            const int dump = cd / prm.n_chan;
            const int c_out = dump * prm.n_chan_total + prm.chan0_out + (cd - dump * prm.n_chan);   // output slab index
            const int r0 = td.row0 + 128 * half;                   // first G row of this CTA
            const int u0 = r0 + quarter * 32;                      // first G row of this warp
            // columns this CTA's rows need: up to the last station of its rows (s_j <= s_i), none for rows past the
            // channel's 2M components
            int need = 0;
            if (r0 < M2) {
                int i_max = (r0 + 127) / (2 * prm.n_pol);
                if (i_max > prm.n_station - 1) i_max = prm.n_station - 1;
                need = (rect ? M2b : (i_max + 1) * 2 * prm.n_pol) - td.col0;
                if (need > kTileCols) need = kTileCols;
                if (need < 0) need = 0;
            }
            const int h_begin = chalf * (kTileCols / 2);
            const int h_end = need < h_begin + kTileCols / 2 ? need : h_begin + kTileCols / 2;
            drain_tile<C::kFloat, true, kPairEpiBufs>(prm, n_kchunks, c_out, u0, td.col0, h_begin, h_end, stage_smem, buf, lane,
                                                      [&](int, uint32_t& taddr, uint32_t& bar) {
                ptx::mbar_wait_uniform(tfull_bar(acc), acc_phase);
                ptx::tc_fence_after();
                taddr = tmem_base + (static_cast<uint32_t>(quarter * 32) << 16) + acc * kTileCols;
                bar = ptx::mapa(tempty_bar(acc), 0);
                if (++acc == 2) { acc = 0; acc_phase ^= 1u; }
            });
        }
        if (lane < 8) ptx::bulk_wait<0>();           // all bulk stores performed before the CTA retires
    }

    // no CTA may exit (or free TMEM) while its peer can still signal its barriers or read its operands
    ptx::tc_fence_before();
    ptx::cluster_sync();
    if (warp == 1) {
        ptx::tc_fence_after();
        ptx::tmem_dealloc_pair(tmem_base, 512);
    }
}

}  // namespace xtc
