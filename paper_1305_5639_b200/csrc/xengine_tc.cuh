// xengine_tc.cuh -- the X-engine as a per-channel Hermitian rank-T update on tcgen05 tensor cores.
//
// Computes PAPER.md:54-57 (Sec. 2, Eq. 2)  V_ij[c] = sum_t conj(x_i[t][c]) x_j[t][c]  for the lower
// station triangle incl. autocorrelations and writes the packed-baseline output.
//
// DIRECT feed ("Gram of components"): for a fixed channel the input is a real matrix
// Y[t][u], u = 2*m + {0: re, 1: im}, m = s*P + p, contiguous in u.  The real Gram matrix
// G = Y^T Y (contraction over time) holds every product Eq. 2 needs:
//     Re V_mn = G[2m][2n]   + G[2m+1][2n+1]
//     Im V_mn = G[2m][2n+1] - G[2m+1][2n]                       (conj on the first index m)
// Both MMA operands are MN-major (u contiguous, K = time strided), so TMA boxes
// [KSTAGE time rows] x [128 bytes of u] are cut straight out of in[t][c][s][p] -- no corner turn,
// no staging copy.  One CTA tile is 128 rows (u) x up to 256 columns (u) of G for one channel;
// the accumulator lives in TMEM (256 columns, double buffered), and the epilogue forms Re/Im with
// one shuffle between adjacent TMEM lanes and streams the packed triangle to HBM.
//
// Warp roles (320 threads, 1 CTA / SM, persistent over a static round-robin of tiles):
//   warp 0      TMA producer  (one elected lane of the converged warp, see ptx::elect_one)
//   warp 1      TMEM allocator + tcgen05.mma issuer (one elected lane)
//   warps 2..9  epilogue: tcgen05.ld -> combine -> shared-memory staging in packed-baseline order ->
//               bulk async store (or bulk reduce-add when accumulating) of whole station-row segments.
//               Warp w owns TMEM lanes 32 (w % 4) .. +31 and the column half (w - 2) / 4 of the tile.
//
// Integration in time is cut into K-chunks of `k_chunk` samples per TMEM accumulation pass: the int8
// path uses one chunk (int32 sums are exact); the fp16 path uses 1024 samples so that the tensor
// core's fp32 accumulator (which truncates when it aligns addends)
// never integrates more than 64 MMAs before its content is folded into the output with an IEEE
// round-to-nearest fp32 add (the L2's reduce-add).  Chunk 0 stores (or reduce-adds if the call
// accumulates), chunks >= 1 reduce-add.
#pragma once
#include "ptx.cuh"

namespace xtc {

constexpr int kMaxStages = 12;                // barrier slots; the stage count is chosen per geometry (Params::n_stages)
constexpr int kRingBytes = 144 * 1024;        // operand ring of the 1-CTA kernel, cut into n_stages stages of stage_bytes
constexpr int kTileRows = 128;        // G rows per tile   (TMEM lanes)
constexpr int kTileCols = 256;        // G columns per tile (TMEM columns per accumulator stage)
constexpr int kNumEpiWarps = 8;
constexpr int kNumThreads = 64 + 32 * kNumEpiWarps;
// epilogue staging (n_pol == 2): one pass = 64 G columns = 16 stations j; a warp's 32 TMEM lanes are
// 8 stations i; one station-row segment is 16 x 32 B = 512 B, padded to 544 B (bank spread, 16-B aligned)
constexpr int kFloatChunk = 1024;   // fp16 path: samples per TMEM accumulation pass
constexpr int kEpiCols = 64;
constexpr int kEpiRowBytes = 544;
constexpr int kEpiBufBytes = 8 * kEpiRowBytes;
constexpr int kEpiWarpBytes = 2 * kEpiBufBytes;                       // double buffered
constexpr int kEpiBytes = kNumEpiWarps * kEpiWarpBytes;
constexpr int kSmemBytes = kRingBytes + kEpiBytes + 1024 /*alignment slack*/ + 256 /*barriers*/;

struct TileDesc {
    int row0;    // first G row   of the tile, in real components u within the channel (multiple of 128)
    int col0;    // first G column of the tile (multiple of 256)
    int ncols;   // columns to compute: multiple of 16, <= 256 (triangular cut and channel edge)
    int pad;
};

struct Params {
    const TileDesc* tiles;   // DEVICE: per-channel tile table
    int tiles_per_chan;
    long long n_tiles;       // tiles_per_chan * n_chan
    int n_station, n_pol, n_chan, n_time;
    int M;                   // n_station * n_pol  (inputs per channel)
    long long n_baseline;    // N(N+1)/2
    void* out;               // DEVICE: packed output
    unsigned long long out_bytes;   // extent of `out`: every bulk store / reduce-add is checked against it (a violation traps)
    int accumulate;
    int k_chunk;             // samples per TMEM accumulation pass (multiple of the pipeline stage)
    // rectangular cross-only mode: rows are the n_station streams of group A (conjugated), columns the
    // n_station_b stations (M_b = n_station_b * n_pol streams) of group B; 0 = triangular HERK of one group
    int n_station_b, M_b;
    // pair kernels: number of separate integrations of n_time samples in one call (corr_xengine_dumps); the input is
    // [n_dump][n_time][C][...], the output [n_dump][C][...]: integration d, channel c is handled as "channel" d*C + c
    int n_dump;
    // channel window (corr_create_window; "separating frequency channels prior to the CMAC stage"): the
    // call integrates n_chan channels starting at channel chan0 of the input (whose row pitch the tensor map carries)
    // into the output slabs chan0_out .. of an output laid out for n_chan_total channels (integration d of a dump call
    // starts at slab d * n_chan_total).  Whole-band plans: 0, 0 and n_chan.
    int chan0, chan0_out, n_chan_total;
    // 1-CTA kernel: a stage holds [b_chunks 128-byte-wide B chunks][A chunks, only if some tile is off the diagonal]
    int n_stages, stage_bytes, b_chunks;
};

template <int kElt> struct Cfg;
template <> struct Cfg<1> {                      // complex int8 -> int32
    static constexpr int kKStage = 128;          // time samples per pipeline stage of the 1-CTA kernel (one TMA box)
    static constexpr int kMmaK = 32;             // time samples per tcgen05.mma (kind::i8)
    static constexpr bool kFloat = false;
    // instruction descriptor: D = S32 (2<<4), A = B = signed 8 bit (1<<7, 1<<10), A and B MN-major
    // (1<<15, 1<<16), M = 128 (8<<24); N is OR-ed in per tile ((N>>3) << 17).
    static constexpr uint32_t kIdesc = (2u << 4) | (1u << 7) | (1u << 10) | (1u << 15) | (1u << 16) | (8u << 24);
};
template <> struct Cfg<2> {                      // complex fp16 -> fp32
    static constexpr int kKStage = 64;
    static constexpr int kMmaK = 16;
    static constexpr bool kFloat = true;
    // D = F32 (1<<4), A = B = F16 (0), MN-major both, M = 128.
    static constexpr uint32_t kIdesc = (1u << 4) | (1u << 15) | (1u << 16) | (8u << 24);
};

template <bool kFloat> __device__ __forceinline__ uint32_t add_bits(uint32_t a, uint32_t b) {
    if constexpr (kFloat) return __float_as_uint(__uint_as_float(a) + __uint_as_float(b));
    else return a + b;
}
template <bool kFloat> __device__ __forceinline__ uint32_t sub_bits(uint32_t a, uint32_t b) {
    if constexpr (kFloat) return __float_as_uint(__uint_as_float(a) - __uint_as_float(b));
    else return a - b;
}

// Re/Im of eight (m, n) products from one 32-column TMEM chunk.  Lane pair (2k, 2k+1) holds G rows
// (2m, 2m+1); columns (2x, 2x+1) are (re, im) of input n0 + x.  On return the even lane (ri = 0) holds
// (re, im) of inputs n0 + 2y, the odd lane of inputs n0 + 2y + 1, y = 0..7.
template <bool kFloat>
__device__ __forceinline__ void combine_chunk(const uint32_t (&v)[32], int ri, uint32_t (&re)[8], uint32_t (&im)[8]) {
    uint32_t w[16];
#pragma unroll
    for (int x = 0; x < 16; ++x) {
        // even lane: Re = G[2m][2n] + G[2m+1][2n+1];  odd lane: Im = G[2m][2n+1] - G[2m+1][2n]
        const uint32_t other = __shfl_xor_sync(0xffffffffu, v[2 * x + 1], 1);
        w[x] = ri ? sub_bits<kFloat>(other, v[2 * x]) : add_bits<kFloat>(v[2 * x], other);
    }
#pragma unroll
    for (int y = 0; y < 8; ++y) {
        const uint32_t send = ri ? w[2 * y] : w[2 * y + 1];
        const uint32_t recv = __shfl_xor_sync(0xffffffffu, send, 1);
        re[y] = ri ? recv : w[2 * y];
        im[y] = ri ? w[2 * y + 1] : recv;
    }
}

// Drain one TMEM accumulator pass of one tile through this epilogue warp: tcgen05.ld -> Re/Im combine ->
// packed-baseline writer (+ accumulate).  The warp owns TMEM lanes [32 quarter, +32) = G rows u0 .. u0 + 31 of
// output slab c (global channel, or integration * n_chan_total + channel) and the tile columns [h_begin, h_end)
// (G columns col0 + h; at most 128 of them); `taddr` addresses lane 32 quarter, column 0 of the accumulator.
// `release_bar` is arrived on (by lane 0; `kRemote`: it lives in the pair leader CTA and is a shared::cluster address)
// as soon as the warp's last TMEM column is in registers.
//
// kFold (fp16 path, several TMEM passes per tile): the passes of one tile are summed in REGISTERS with IEEE
// round-to-nearest fp32 adds and only the last pass touches memory:
//   kFoldNone  single pass: combine -> stage -> store / reduce-add
//   kFoldAdd   run[] += this pass; nothing is written
//   kFoldLast  this pass + run[] -> stage -> store / reduce-add
// run[k]: the warp's (re, im) values in the order they are produced: 32-column chunk q (0..3), then re[0..7], im[0..7].
enum { kFoldNone = 0, kFoldAdd = 1, kFoldLast = 2 };

template <bool kFloat, int kFold>
__device__ __forceinline__ void fold_chunk(uint32_t (&re)[8], uint32_t (&im)[8], float (&run)[64], int q) {
    if constexpr (kFloat && kFold != kFoldNone) {
#pragma unroll
        for (int y = 0; y < 8; ++y) {
            const float r = __uint_as_float(re[y]) + run[q * 16 + y];
            const float i = __uint_as_float(im[y]) + run[q * 16 + 8 + y];
            if constexpr (kFold == kFoldAdd) {
                run[q * 16 + y] = r;
                run[q * 16 + 8 + y] = i;
            } else {
                re[y] = __float_as_uint(r);
                im[y] = __float_as_uint(i);
            }
        }
    }
}

template <bool kFloat, bool kRemote, int kBufs, int kFold>
__device__ __forceinline__ void drain_accumulator(const Params& prm, int c, int u0, int col0, int h_begin, int h_end,
                                                  uint32_t taddr, uint32_t release_bar, bool reduce,
                                                  uint32_t stage_smem, int& buf, int lane, float (&run)[64]) {
    auto release = [&]() {
        ptx::tc_fence_before();
        __syncwarp();
        if (lane == 0) {
            if constexpr (kRemote) ptx::mbar_arrive_cluster(release_bar);
            else ptx::mbar_arrive(release_bar);
        }
    };
    const int P = prm.n_pol;
    const int ri = lane & 1;                     // row parity: 0 = re row (u even), 1 = im row
    uint8_t* out8 = static_cast<uint8_t*>(prm.out);
    const bool rect = prm.n_station_b > 0;
    const uint64_t policy = ptx::policy_evict_first();
    if (h_begin >= h_end) {                      // nothing in this column half: just release
        release();
        return;
    }
    if (P == 2) {
        // ---- fast path: station rows are 32-byte aligned runs; bulk async store / reduce-add ----
        const int il = lane >> 2;                        // station within the warp's 8
        const int p = (lane >> 1) & 1;
        const int i_row = (u0 >> 2) + lane;              // lanes 0..7: the station row this lane ships
#pragma unroll
        for (int it = 0; it < (kTileCols / 2) / kEpiCols; ++it) {
            const int h0 = h_begin + it * kEpiCols;
            if (h0 >= h_end) continue;                   // (no break: the loop must unroll so that run[] stays in registers)
            const uint32_t sbuf = stage_smem + buf * kEpiBufBytes;
            if constexpr (kFold != kFoldAdd) {
                if (lane < 8) ptx::bulk_wait_read<kBufs - 1>();   // staging[buf] (kBufs passes ago) has been read
                __syncwarp();
            }
            const bool two = h0 + 32 < h_end;
            if constexpr (kFold == kFoldNone) {
                // both 32-column TMEM loads of the pass are issued before the first wait (latency overlap)
                uint32_t v0[32], v1[32];
                ptx::tmem_ld_32x32(taddr + h0, v0);
                if (two) ptx::tmem_ld_32x32(taddr + h0 + 32, v1);
                ptx::tmem_ld_wait();
                if (h0 + kEpiCols >= h_end) release();       // all of this warp's columns are in registers
                {
                    uint32_t re[8], im[8];
                    combine_chunk<kFloat>(v0, ri, re, im);
                    // (i, p) x (j = j0 + 8 half + y, q = ri): byte offset j*32 + p*16 + q*8 in the station row
                    const uint32_t dst = sbuf + il * kEpiRowBytes + p * 16 + ri * 8;
#pragma unroll
                    for (int y = 0; y < 8; ++y) ptx::st_shared_v2(dst + y * 32, re[y], im[y]);
                }
                if (two) {
                    uint32_t re[8], im[8];
                    combine_chunk<kFloat>(v1, ri, re, im);
                    const uint32_t dst = sbuf + il * kEpiRowBytes + 256 + p * 16 + ri * 8;
#pragma unroll
                    for (int y = 0; y < 8; ++y) ptx::st_shared_v2(dst + y * 32, re[y], im[y]);
                }
            } else {
                // folding passes keep 64 running sums per thread: one 32-column chunk at a time (register budget: 168)
#pragma unroll
                for (int q = 0; q < 2; ++q) {
                    if (q == 1 && !two) continue;
                    uint32_t v[32];
                    ptx::tmem_ld_32x32(taddr + h0 + 32 * q, v);
                    ptx::tmem_ld_wait();
                    if (h0 + 32 * (q + 1) >= h_end) release();
                    uint32_t re[8], im[8];
                    combine_chunk<kFloat>(v, ri, re, im);
                    fold_chunk<kFloat, kFold>(re, im, run, 2 * it + q);
                    if constexpr (kFold == kFoldLast) {
                        const uint32_t dst = sbuf + il * kEpiRowBytes + 256 * q + p * 16 + ri * 8;
#pragma unroll
                        for (int y = 0; y < 8; ++y) ptx::st_shared_v2(dst + y * 32, re[y], im[y]);
                    }
                }
            }
            if constexpr (kFold != kFoldAdd) {
                ptx::fence_proxy_async_smem();               // generic-proxy writes -> visible to the bulk copy
                __syncwarp();
                if (lane < 8) {
                    const int j0 = (col0 + h0) >> 2;                          // first station of this pass
                    int cnt = (h_end - h0) >> 2;                              // stations staged in this pass
                    if (cnt > kEpiCols / 4) cnt = kEpiCols / 4;
                    const int j_end = rect ? prm.n_station_b : i_row + 1;     // triangle: j <= i; rectangle: every j of group B
                    if (cnt > j_end - j0) cnt = j_end - j0;
                    if (i_row < prm.n_station && cnt > 0) {
                        const long long row = rect ? (static_cast<long long>(c) * prm.n_station + i_row) * prm.n_station_b
                                                   : static_cast<long long>(c) * prm.n_baseline + static_cast<long long>(i_row) * (i_row + 1) / 2;
                        uint8_t* dst = out8 + ((row + j0) << 5);
                        const uint32_t src = sbuf + lane * kEpiRowBytes;
                        const uint32_t bytes = static_cast<uint32_t>(cnt) << 5;
                        // the writer's own bounds check (compute-sanitizer is not available on every box): a segment
                        // outside the caller's buffer or the warp's staging row is a bug, never a silent write
                        if (((row + j0) << 5) < 0 || static_cast<unsigned long long>((row + j0) << 5) + bytes > prm.out_bytes ||
                            bytes > static_cast<uint32_t>(kEpiRowBytes)) __trap();
                        if (!reduce) ptx::bulk_store(dst, src, bytes, policy);
                        else if constexpr (kFloat) ptx::bulk_reduce_add_f32(dst, src, bytes, policy);
                        else ptx::bulk_reduce_add_s32(dst, src, bytes, policy);
                    }
                    ptx::bulk_commit();
                }
                if (kBufs == 2) buf ^= 1;
            }
        }
    } else {
        // ---- general path (n_pol == 1): per-visibility 8-byte stores ----
        const int m = (u0 + lane) >> 1;                  // conjugated input of this lane pair
        const int i = m / P, p = m - i * P;
        const bool row_ok = m < prm.M;
        // word offset of (c, b(i,0), p, q=0); b(i,j) = i(i+1)/2 + j
        const long long row = rect ? (static_cast<long long>(c) * prm.n_station + i) * prm.n_station_b
                                   : static_cast<long long>(c) * prm.n_baseline + static_cast<long long>(i) * (i + 1) / 2;
        const long long row_base = (row * P + p) * P * 2;
        const int n_cols = rect ? prm.M_b : prm.M;
        uint32_t* out = static_cast<uint32_t*>(prm.out);
#pragma unroll
        for (int it = 0; it < (kTileCols / 2) / 32; ++it) {
            const int h0 = h_begin + it * 32;
            if (h0 >= h_end) continue;
            uint32_t v[32];
            ptx::tmem_ld_32x32(taddr + h0, v);
            ptx::tmem_ld_wait();
            if (h0 + 32 >= h_end) release();
            uint32_t re[8], im[8];
            combine_chunk<kFloat>(v, ri, re, im);
            fold_chunk<kFloat, kFold>(re, im, run, it);
            if constexpr (kFold != kFoldAdd) {
                const int n0 = (col0 + h0) >> 1;
#pragma unroll
                for (int y = 0; y < 8; ++y) {
                    const int n = n0 + 2 * y + ri;
                    const int j = n / P, q = n - j * P;
                    if (row_ok && n < n_cols && (rect || j <= i)) {
                        const long long word = row_base + (static_cast<long long>(j) * P * P + q) * 2;
                        if (word < 0 || static_cast<unsigned long long>(word + 2) * 4 > prm.out_bytes) __trap();
                        uint2* dst = reinterpret_cast<uint2*>(out + word);
                        uint2 val = make_uint2(re[y], im[y]);
                        if (reduce) {
                            const uint2 old = *dst;
                            val.x = add_bits<kFloat>(old.x, val.x);
                            val.y = add_bits<kFloat>(old.y, val.y);
                        }
                        *dst = val;
                    }
                }
            }
        }
    }
}

// All TMEM passes of one tile through this epilogue warp (see drain_accumulator): `wait_pass(kc)` blocks until pass kc
// of the tile is complete in TMEM and returns {TMEM address, release barrier} of the accumulator it sits in.
template <bool kFloat, bool kRemote, int kBufs, typename WaitPass>
__device__ __forceinline__ void drain_tile(const Params& prm, int n_kchunks, int c, int u0, int col0, int h_begin, int h_end,
                                           uint32_t stage_smem, int& buf, int lane, WaitPass&& wait_pass) {
    float run[64];
    const bool acc = prm.accumulate != 0;
    if (!kFloat || n_kchunks == 1) {
        for (int kc = 0; kc < n_kchunks; ++kc) {          // int32: one pass by construction
            uint32_t taddr, bar;
            wait_pass(kc, taddr, bar);
            drain_accumulator<kFloat, kRemote, kBufs, kFoldNone>(prm, c, u0, col0, h_begin, h_end, taddr, bar, acc || kc != 0,
                                                                 stage_smem, buf, lane, run);
        }
        return;
    }
    if constexpr (kFloat) {
#pragma unroll
        for (int k = 0; k < 64; ++k) run[k] = 0.0f;
        for (int kc = 0; kc < n_kchunks; ++kc) {
            uint32_t taddr, bar;
            wait_pass(kc, taddr, bar);
            if (kc + 1 < n_kchunks)
                drain_accumulator<kFloat, kRemote, kBufs, kFoldAdd>(prm, c, u0, col0, h_begin, h_end, taddr, bar, false, stage_smem,
                                                                    buf, lane, run);
            else
                drain_accumulator<kFloat, kRemote, kBufs, kFoldLast>(prm, c, u0, col0, h_begin, h_end, taddr, bar, acc, stage_smem,
                                                                     buf, lane, run);
        }
    }
}

template <int kElt>
__global__ void __launch_bounds__(kNumThreads, 1)
xengine_direct_kernel(const __grid_constant__ CUtensorMap tmap_in, const Params prm) {
    using C = Cfg<kElt>;
    constexpr int kChunkElems = 128 / kElt;                 // u per 128-byte chunk
    constexpr int kChunkBytes = C::kKStage * 128;           // one TMA box: [KSTAGE rows][128 B]
    constexpr int kAChunks = kTileRows / kChunkElems;       // 1 (ci8) / 2 (cf16)
    constexpr int kBChunksMax = kTileCols / kChunkElems;    // 2 (ci8) / 4 (cf16)
    constexpr int kKStepBytes = C::kMmaK * 128;             // smem advance per MMA k-step
    constexpr int kKSteps = C::kKStage / C::kMmaK;          // 4
    static_assert((kAChunks + kBChunksMax) * kChunkBytes * 3 <= kRingBytes, "at least three stages");
    const int kNumStages = prm.n_stages;
    const int kStageBytes = prm.stage_bytes;

    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;   // SWIZZLE_128B atoms: 1024-B aligned
    const uint32_t epi_base = smem_base + kRingBytes;
    const uint32_t bar_base = epi_base + kEpiBytes;
    // barrier slots (8 bytes each): full[S], empty[S], tmem_full[2], tmem_empty[2], then the TMEM base word
    auto full_bar = [&](int s) { return bar_base + 8u * s; };
    auto empty_bar = [&](int s) { return bar_base + 8u * (kMaxStages + s); };
    auto tfull_bar = [&](int a) { return bar_base + 8u * (2 * kMaxStages + a); };
    auto tempty_bar = [&](int a) { return bar_base + 8u * (2 * kMaxStages + 2 + a); };
    const uint32_t tmem_slot = bar_base + 8u * (2 * kMaxStages + 4);
    uint32_t* tmem_slot_ptr =
        reinterpret_cast<uint32_t*>(smem_raw + (tmem_slot - ptx::smem_u32(smem_raw)));

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;

    if (threadIdx.x == 0) {
        ptx::prefetch_tensormap(&tmap_in);
        for (int s = 0; s < kNumStages; ++s) {
            ptx::mbar_init(full_bar(s), 1);
            ptx::mbar_init(empty_bar(s), 1);
        }
        for (int a = 0; a < 2; ++a) {
            ptx::mbar_init(tfull_bar(a), 1);
            ptx::mbar_init(tempty_bar(a), kNumEpiWarps);      // one arrive per epilogue warp
        }
        ptx::fence_mbar_init();
    }
    if (warp == 1) {
        ptx::tmem_alloc(tmem_slot, 512);
        ptx::tmem_relinquish();
    }
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_ptr;

    const int num_kb = (prm.n_time + C::kKStage - 1) / C::kKStage;     // pipeline stages over the whole integration
    const int kb_per_chunk = prm.k_chunk / C::kKStage > 0 ? prm.k_chunk / C::kKStage : 1;
    const int n_kchunks = (num_kb + kb_per_chunk - 1) / kb_per_chunk;
    const int M2 = 2 * prm.M;

    if (warp == 0) {
        // ===================== TMA producer (whole warp in uniform control flow, one elected lane issues) =====================
        {
            int stage = 0;
            uint32_t phase = 0;
            for (long long tile = blockIdx.x; tile < prm.n_tiles; tile += gridDim.x) {
                const int c = static_cast<int>(tile / prm.tiles_per_chan);
                const TileDesc* tdp = prm.tiles + (tile - static_cast<long long>(c) * prm.tiles_per_chan);
                const int row0 = static_cast<int>(ptx::uniform(tdp->row0)), col0 = static_cast<int>(ptx::uniform(tdp->col0));
                const int ncols = static_cast<int>(ptx::uniform(tdp->ncols));
                const int w_row = (prm.chan0 + c) * M2 + row0;           // element coordinate in the [T][C*2M] view
                const int w_col = (prm.chan0 + c) * M2 + col0;
                const int nb = (ncols + kChunkElems - 1) / kChunkElems;
                // tile on the diagonal: the 128 A rows are among the loaded B columns -> A is not loaded at all
                const bool a_in_b = row0 >= col0 && row0 + kTileRows <= col0 + nb * kChunkElems;
                const uint32_t tx = static_cast<uint32_t>(((a_in_b ? 0 : kAChunks) + nb) * kChunkBytes);
                for (int kb = 0; kb < num_kb; ++kb) {
                    ptx::mbar_wait_uniform(empty_bar(stage), phase ^ 1u);
                    const uint32_t sb = smem_base + stage * kStageBytes;
                    const uint32_t sa = sb + prm.b_chunks * kChunkBytes;
                    if (ptx::elect_one()) {
                        ptx::mbar_arrive_expect_tx(full_bar(stage), tx);
#pragma unroll
                        for (int a = 0; a < kAChunks; ++a)
                            if (!a_in_b)
                                ptx::tma_load_3d(sa + a * kChunkBytes, &tmap_in, full_bar(stage),
                                                 w_row + a * kChunkElems, kb * C::kKStage, 0);
#pragma unroll
                        for (int b = 0; b < kBChunksMax; ++b)
                            if (b < nb)
                                ptx::tma_load_3d(sb + b * kChunkBytes, &tmap_in, full_bar(stage),
                                                 w_col + b * kChunkElems, kb * C::kKStage, 0);
                    }
                    __syncwarp();
                    if (++stage == kNumStages) { stage = 0; phase ^= 1u; }
                }
            }
        }
    } else if (warp == 1) {
        // ===================== MMA issuer (whole warp in uniform control flow, one elected lane issues) =====================
        {
            const uint32_t tb = ptx::uniform(tmem_base);
            int stage = 0;
            uint32_t phase = 0;
            int acc = 0;
            uint32_t acc_phase = 0;
            for (long long tile = blockIdx.x; tile < prm.n_tiles; tile += gridDim.x) {
                const int c = static_cast<int>(tile / prm.tiles_per_chan);
                const TileDesc* tdp = prm.tiles + (tile - static_cast<long long>(c) * prm.tiles_per_chan);
                const int row0 = static_cast<int>(ptx::uniform(tdp->row0)), col0 = static_cast<int>(ptx::uniform(tdp->col0));
                const int ncols = static_cast<int>(ptx::uniform(tdp->ncols));
                const uint32_t idesc = C::kIdesc | (static_cast<uint32_t>(ncols >> 3) << 17);
                const int nb = (ncols + kChunkElems - 1) / kChunkElems;
                const bool a_in_b = row0 >= col0 && row0 + kTileRows <= col0 + nb * kChunkElems;
                // A operand = the B chunks holding rows row0 .. row0 + 127 when the tile lies on the diagonal
                const uint32_t a_off = (a_in_b ? (row0 - col0) / kChunkElems : prm.b_chunks) * kChunkBytes;
                for (int kb0 = 0; kb0 < num_kb; kb0 += kb_per_chunk) {
                    const int kb1 = kb0 + kb_per_chunk < num_kb ? kb0 + kb_per_chunk : num_kb;
                    const uint32_t d_tmem = tb + acc * kTileCols;
                    ptx::mbar_wait_uniform(tempty_bar(acc), acc_phase ^ 1u);     // epilogue has drained this accumulator
                    ptx::tc_fence_after();
                    for (int kb = kb0; kb < kb1; ++kb) {
                        ptx::mbar_wait_uniform(full_bar(stage), phase);          // TMA bytes have landed
                        ptx::tc_fence_after();
                        const uint32_t sb = smem_base + stage * kStageBytes;
                        if (ptx::elect_one()) {
#pragma unroll
                            for (int k = 0; k < kKSteps; ++k) {
                                // MN-major SWIZZLE_128B: LBO = distance between 128-byte-wide chunks (one TMA box),
                                // SBO = distance between 8-row groups along K (8 * 128 B).
                                const uint64_t adesc = ptx::smem_desc_sw128(sb + a_off + k * kKStepBytes, kChunkBytes, 1024);
                                const uint64_t bdesc = ptx::smem_desc_sw128(sb + k * kKStepBytes, kChunkBytes, 1024);
                                const uint32_t accum = (kb != kb0 || k != 0) ? 1u : 0u;
                                if constexpr (C::kFloat) ptx::mma_f16(d_tmem, adesc, bdesc, idesc, accum);
                                else ptx::mma_i8(d_tmem, adesc, bdesc, idesc, accum);
                            }
                            ptx::mma_commit(empty_bar(stage));               // frees the smem slot when the MMAs retire
                            if (kb + 1 == kb1) ptx::mma_commit(tfull_bar(acc));   // accumulator complete -> epilogue
                        }
                        __syncwarp();
                        if (++stage == kNumStages) { stage = 0; phase ^= 1u; }
                    }
                    if (++acc == 2) { acc = 0; acc_phase ^= 1u; }
                }
            }
        }
    } else {
        // ===================== epilogue: combine + packed-baseline writer =====================
        const int ew = warp - 2;
        const int quarter = warp & 3;                // TMEM lanes [32*quarter, 32*quarter+32) belong to this warp
        const int chalf = ew >> 2;                   // column half of the tile handled by this warp
        const uint32_t stage_smem = epi_base + ew * kEpiWarpBytes;
        int acc = 0;
        uint32_t acc_phase = 0;
        int buf = 0;
        for (long long tile = blockIdx.x; tile < prm.n_tiles; tile += gridDim.x) {
            const int c = static_cast<int>(tile / prm.tiles_per_chan);
            const TileDesc td = prm.tiles[tile - static_cast<long long>(c) * prm.tiles_per_chan];
            const int u0 = td.row0 + quarter * 32;                 // first G row of this warp
            const int h_begin = chalf * (kTileCols / 2);
            const int h_end = td.ncols < h_begin + kTileCols / 2 ? td.ncols : h_begin + kTileCols / 2;
            drain_tile<C::kFloat, false, 2>(prm, n_kchunks, prm.chan0_out + c, u0, td.col0, h_begin, h_end, stage_smem, buf, lane,
                                            [&](int, uint32_t& taddr, uint32_t& bar) {
                ptx::mbar_wait_uniform(tfull_bar(acc), acc_phase);
                ptx::tc_fence_after();
                taddr = tmem_base + (static_cast<uint32_t>(quarter * 32) << 16) + acc * kTileCols;
                bar = tempty_bar(acc);
                if (++acc == 2) { acc = 0; acc_phase ^= 1u; }
            });
        }
        if (lane < 8) ptx::bulk_wait<0>();           // all bulk stores performed before the CTA retires
    }

    ptx::tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        ptx::tc_fence_after();
        ptx::tmem_dealloc(tmem_base, 512);
    }
}

}  // namespace xtc
