// fengine_tc.cuh -- the F-engine as a dense contraction on tcgen05 tensor cores.
//
// PAPER.md:49-52 (Sec. 2, Eq. 1):  S[k] = sum_{n=0}^{N-1} s[n] exp(-j (2 pi / N) k n),  N = 256, on
// consecutive blocks of every stream's 8-bit REAL samples.  For real input the sum folds onto n = 0 .. 128:
//     e[0] = s[0],  e[n] = s[n] + s[256 - n],  o[n] = s[n] - s[256 - n]      (n = 1 .. 127; integers, exact in fp16)
//     Re S[k] =  sum_{n=0}^{127} e[n] cos(2 pi k n / 256)  +  (-1)^k s[128]
//     Im S[k] = -sum_{n=1}^{127} o[n] sin(2 pi k n / 256)
// i.e. two [128 folded samples] x [128 channels] matrices applied to the folded samples of every (stream, spectrum): a GEMM
// with M = 128 (stream, spectrum) rows, K = 128 (folded samples), N = 128 (channels).  The twiddle matrices are split into
// fp16 hi + lo parts (cos = hi + lo to ~3e-8 absolute), every product e * hi, e * lo is exact in the fp32 accumulator,
// so the result carries only the accumulation round-off: well inside the fp32 bound the parity test allows
// (0.5 ulp of the fp16 output + 2e-6 sum|s|).  The slot o[0] (whose sine is zero) carries s[128], and one extra k-step
// against a matrix that is (-1)^k in that slot and zero elsewhere adds the Nyquist term to Re, exactly.
//
// Orientation (third version; measurements in DESIGN.md 5.6): rows of the accumulator are STREAMS, columns are CHANNELS.
//  * The A operand -- the folded samples of the tile -- is written straight into TENSOR MEMORY by the fold warps
//    (tcgen05.st, one row per thread) and never touches shared memory; B -- the four twiddle matrices, 128 KB -- stays
//    resident in shared memory for the whole kernel.
//  * The epilogue needs no transpose: a warp's 32 TMEM lanes are 32 consecutive streams, so for every channel the warp
//    stores one full 128-byte line of the X-engine's [spectrum][channel][stream] layout straight from registers.
//  The first tensor-core version (twiddles as A in TMEM, samples as B through shared memory, transposing epilogue) moved
//  ~190 KB through shared memory per 64 streams and was bound by that (83 % of the 128 B/clk pipe with all global traffic
//  removed); this one moves ~96 KB, half of it the MMAs' own B reads.
//
// One CTA (cta_group::1, 576 threads, persistent over tiles of two half tiles = 2 x (64 streams of one spectrum)):
//   warp 0      TMA: raw int8 half tiles [64 streams][256 samples] (two SWIZZLE_128B boxes) into a 5-deep ring
//   warp 1      tcgen05.mma issuer (one elected lane, uniform control flow): per tile 17 MMAs (M 128, N 128, K 16) into the
//               Re accumulator and 16 into the Im accumulator; the two accumulators are handed to the epilogue separately,
//               so Re of tile t drains while Im of tile t is computed, and Im drains under Re of tile t + 1
//   warps 2-9   fold + convert: raw int8 -> e, o as fp16 (bytes become halves with the 0x6400 | byte trick, no
//               integer-to-float conversion instruction) -> tcgen05.st into the A buffer (double buffered);
//               thread = one stream row, two warps per TMEM lane quarter split the sample groups
//   warps 10-17 epilogue: two warps per lane quarter, 64 channels each: Re -> packed halves in registers, then Im ->
//               (re, im) half2 words -> one coalesced 128-byte store per channel and warp.  kInt8 (corr_fengine_ci8):
//               requantised (re, im) int8 codes instead; the two warps of a half tile trade halves through an exchange
//               buffer so that the stores are still full 128-byte lines (4-deep raw ring, the fifth slot is the buffers)
#pragma once
#include <cuda_fp16.h>
#include <type_traits>
#include "ptx.cuh"

namespace fengtc {

constexpr int kFft = 256;
constexpr int kChan = 128;                    // channels kept = MMA N
constexpr int kFold = 128;                    // folded samples = GEMM K
constexpr int kTileStreams = 64;              // streams of one half tile (a ragged last one: TMA zero-fills, stores are predicated)
constexpr int kFoldWarps = 8, kEpiWarps = 8;
constexpr int kThreads = 64 + 32 * (kFoldWarps + kEpiWarps);
constexpr int kRawBytes = kTileStreams * kFft;               // one half tile: 16 KB (two boxes of 64 rows x 128 B)
constexpr int kRawRing = 5;                                  // half tiles in flight per CTA (fp16 output)
// int8 output: 4 half tiles, the fifth slot is the epilogue's exchange buffer: a warp's 32 streams are only 64 bytes of an
// int8 output row, and the write path is bound by the number of line requests, not by bytes (measured: 64-byte stores
// took as long as the fp16 kernel's 128-byte stores), so the two warps of a half tile assemble full 128-byte lines
constexpr int kRawRingI8 = 4;
constexpr int kXchgBytes = 32 * 128;                         // per warp pair: 32 channels x 64 streams x (re, im) int8
constexpr int kMatBytes = kChan * kFold * 2;                 // one fp16 twiddle matrix: 32 KB (two K chunks of 16 KB)
constexpr int kNumMats = 5;                                  // cos_hi, cos_lo, -sin_hi, -sin_lo, Nyquist sign (first K chunk only)
// tensor memory map (columns): Re accumulator, Im accumulator, two A buffers {e: 64 columns, o: 64 columns}
constexpr int kTmemRe = 0, kTmemIm = 128, kTmemA = 256, kTmemABuf = 128, kTmemCols = 512;
// shared memory map (offsets from the 1024-byte aligned base)
constexpr int kOffTw = 0;
constexpr int kOffNyq = 4 * kMatBytes;                       // 16 KB
constexpr int kOffRaw = kOffNyq + kMatBytes / 2;
constexpr int kOffBar = kOffRaw + kRawRing * kRawBytes;
constexpr int kSmemBytes = kOffBar + 256 + 1024 /*alignment slack*/;
static_assert(kSmemBytes <= 227 * 1024, "shared memory");

struct Params {
    void* out;               // [n_spectra][128][n_stream] __half2 (re, im); kInt8: char2 codes clip(rint(S * scale), +-127)
    float scale;             // kInt8 only
    const uint4* tw;         // DEVICE: twiddles [cos_hi | cos_lo | -sin_hi | -sin_lo | nyquist][128 channels][128 samples] fp16
    int n_stream;            // multiple of 64
    long long n_spectra;
    long long n_half;        // half tiles: n_spectra * ceil(n_stream / 64)
    long long n_tiles;       // (n_half + 1) / 2
};

// instruction descriptor: D = F32 (1 << 4), A = B = F16, both K-major, M = 128 (8 << 24), N = 128 (16 << 17)
constexpr uint32_t kIdesc = (1u << 4) | (8u << 24) | (static_cast<uint32_t>(kChan >> 3) << 17);

__device__ __forceinline__ uint32_t lds_u32(uint32_t addr) {
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ uint4 lds_v4(uint32_t addr) {
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
    return v;
}
__device__ __forceinline__ void sts_v4(uint32_t addr, uint4 v) {
    asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
__device__ __forceinline__ uint32_t hadd2(uint32_t a, uint32_t b) {
    uint32_t d;
    asm("add.rn.f16x2 %0, %1, %2;" : "=r"(d) : "r"(a), "r"(b));
    return d;
}
__device__ __forceinline__ uint32_t hsub2(uint32_t a, uint32_t b) {
    uint32_t d;
    asm("sub.rn.f16x2 %0, %1, %2;" : "=r"(d) : "r"(a), "r"(b));
    return d;
}
// four int8 samples (one 32-bit word) -> two half2 {s0, s1}, {s2, s3}, exact: the byte b of x ^ 0x80 is s + 128 in
// [0, 255]; 0x6400 | b reads as the half 1024 + b; subtracting 1152 leaves s
__device__ __forceinline__ void bytes_to_half2(uint32_t w, uint32_t& lo, uint32_t& hi) {
    const uint32_t x = w ^ 0x80808080u;
    lo = hadd2(__byte_perm(x, 0x64646464u, 0x4140), 0xE480E480u);      // -1152 = 0xE480
    hi = hadd2(__byte_perm(x, 0x64646464u, 0x4342), 0xE480E480u);
}
// two floats -> half2 word {low 16 bits: lo, high 16 bits: hi}, round to nearest even
__device__ __forceinline__ uint32_t pack_half2(float lo, float hi) {
    uint32_t d;
    asm("cvt.rn.f16x2.f32 %0, %1, %2;" : "=r"(d) : "f"(hi), "f"(lo));
    return d;
}
// streaming store of one output word: written once, not read by this kernel: no L1 allocation, first in line for L2 eviction
__device__ __forceinline__ void stg_stream(uint32_t* p, uint32_t v, uint64_t policy) {
    asm volatile("st.global.L1::no_allocate.L2::cache_hint.b32 [%0], %1, %2;" ::"l"(p), "r"(v), "l"(policy) : "memory");
}
// two accumulator values -> one packed pair: fp16 output: half2 word; int8 output (corr_fengine_ci8): the codes
// clip(rint(v * scale), -127, 127) (rint: ties to even; -128 is never produced) in bytes 0 and 1
template <bool kInt8> __device__ __forceinline__ uint32_t pack_pair(float lo, float hi, float scale) {
    if constexpr (kInt8) {
        // No float-to-int instruction (a quarter-rate pipe: 128 of them per thread and tile made this epilogue the slowest
        // stage of the kernel).  ONE fused multiply-add forms v * scale + 1.5 * 2^23 with a single rounding, to nearest even
        // at unit spacing: the float's bit pattern is then 0x4B400000 + rint(v * scale) (two's complement in the mantissa),
        // exact rint of the UNROUNDED product.  The clip to +-127 is taken on those bits as signed integers, which order like
        // the floats they encode (anything beyond +-2^22, where the spacing is no longer 1, lands outside the window on the
        // right side; negative floats are negative integers), and the code is the low byte.
        constexpr int kMagicBits = 0x4B400000;
        const int a = min(max(__float_as_int(fmaf(lo, scale, 12582912.0f)), kMagicBits - 127), kMagicBits + 127);
        const int b = min(max(__float_as_int(fmaf(hi, scale, 12582912.0f)), kMagicBits - 127), kMagicBits + 127);
        return __byte_perm(static_cast<uint32_t>(a), static_cast<uint32_t>(b), 0x0040);     // bytes 0, 1: the two codes
    } else {
        return pack_half2(lo, hi);
    }
}
__device__ __forceinline__ void sts_u16(uint32_t addr, uint32_t v) {
    asm volatile("st.shared.u16 [%0], %1;" ::"r"(addr), "h"(static_cast<uint16_t>(v)) : "memory");
}
// named barrier of one warp pair (64 threads); ids 1 .. 4
__device__ __forceinline__ void pair_sync(int id) { asm volatile("bar.sync %0, 64;" ::"r"(id) : "memory"); }
// a half tile in the raw ring (two SWIZZLE_128B boxes of [64 rows][128 bytes]): 16-byte unit u of row r of box b
__device__ __forceinline__ uint32_t raw_unit(uint32_t slot_base, int b, int r, int u) {
    return slot_base + b * (kRawBytes / 2) + r * 128 + ((u ^ (r & 7)) << 4);
}

// kRagged: n_stream is not a multiple of 64 -- the last half tile of every spectrum is partly beyond the tensor map and the
// epilogue's stores are predicated.  A separate instantiation: the predicates cost the whole-tile kernel 6 % (fp16 output)
// to 11 % (int8 output, a register spill) when they were compiled in unconditionally.
template <bool kInt8, bool kRagged>
__global__ void __launch_bounds__(kThreads, 1)
fengine_tc_kernel(const __grid_constant__ CUtensorMap tmap_raw, const Params prm) {
    extern __shared__ uint8_t smem_raw[];
    const uint32_t base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t bar = base + kOffBar;
    // barriers: raw_full[5], raw_empty[5], a_full[2], a_empty[2], re_full, re_empty, im_full, im_empty, then the TMEM base word
    constexpr int kRing = kInt8 ? kRawRingI8 : kRawRing;
    static_assert(!kInt8 || 4 * kXchgBytes <= (kRawRing - kRawRingI8) * kRawBytes, "exchange buffers");
    const uint32_t raw_full0 = bar, raw_empty0 = raw_full0 + 8 * kRawRing, a_full0 = raw_empty0 + 8 * kRawRing, a_empty0 = a_full0 + 16;
    const uint32_t re_full = a_empty0 + 16, re_empty = re_full + 8, im_full = re_empty + 8, im_empty = im_full + 8;
    const uint32_t tmem_slot = im_empty + 8;
    static_assert(16 * kRawRing + 32 + 32 + 4 <= 256, "barrier region");
    uint32_t* tmem_slot_ptr = reinterpret_cast<uint32_t*>(smem_raw + (tmem_slot - ptx::smem_u32(smem_raw)));

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;

    if (threadIdx.x == 0) {
        ptx::prefetch_tensormap(&tmap_raw);
        for (int k = 0; k < kRing; ++k) {
            ptx::mbar_init(raw_full0 + 8 * k, 1);
            ptx::mbar_init(raw_empty0 + 8 * k, kFoldWarps / 2);   // the four fold warps of the half tile's two lane quarters
        }
        for (int k = 0; k < 2; ++k) {
            ptx::mbar_init(a_full0 + 8 * k, kFoldWarps);
            ptx::mbar_init(a_empty0 + 8 * k, 1);
        }
        ptx::mbar_init(re_full, 1);
        ptx::mbar_init(re_empty, kEpiWarps);
        ptx::mbar_init(im_full, 1);
        ptx::mbar_init(im_empty, kEpiWarps);
        ptx::fence_mbar_init();
    }
    if (warp == 1) {
        ptx::tmem_alloc(tmem_slot, kTmemCols);
        ptx::tmem_relinquish();
    }
    // the twiddle matrices into shared memory, once, in the K-major SWIZZLE_128B layout of a B operand: matrix m, K chunk
    // (64 samples = 128 bytes per channel row), 8-row groups of 1024 bytes, 16-byte units XOR-ed with the row within the group
    for (int idx = threadIdx.x; idx < 4 * kChan * 16 + kChan * 8; idx += kThreads) {
        const bool nyq = idx >= 4 * kChan * 16;
        const int e = nyq ? idx - 4 * kChan * 16 : idx;
        const int m = nyq ? 4 : e >> 11, k = nyq ? e >> 3 : (e >> 4) & (kChan - 1), u = nyq ? e & 7 : e & 15;
        const uint4 v = __ldg(prm.tw + (m * kChan + k) * (kFold * 2 / 16) + u);
        sts_v4(base + kOffTw + m * kMatBytes + (u >> 3) * (kMatBytes / 2) + (k >> 3) * 1024 + (k & 7) * 128 + (((u & 7) ^ (k & 7)) << 4), v);
    }
    ptx::fence_proxy_async_smem();                           // generic-proxy writes -> visible to the tensor core
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_ptr;

    // half tiles per spectrum (consecutive half tiles share a spectrum).  The last one may be ragged: the tensor map ends at
    // n_stream, so TMA zero-fills the rows beyond it (the full box still counts on the barrier), the fold and the MMAs run on
    // zeros there, and the epilogue stores only streams < n_stream.
    const int n_sb = (prm.n_stream + kTileStreams - 1) / kTileStreams;
    const long long first = blockIdx.x, step = gridDim.x;

    if (warp == 0) {
        // ===================== TMA producer (one elected lane of the converged warp) =====================
        long long pos = 0;                                   // half tiles loaded so far: ring slot pos % 5
        for (long long t = first; t < prm.n_tiles; t += step) {
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const long long hidx = 2 * t + h;
                if (hidx >= prm.n_half) continue;            // odd number of half tiles: the last tile has one
                const long long a = hidx / n_sb;
                const int m0 = static_cast<int>(hidx - a * n_sb) * kTileStreams;
                const int slot = static_cast<int>(pos % kRing);
                const uint32_t phase = static_cast<uint32_t>(pos / kRing) & 1u;
                ptx::mbar_wait_uniform(raw_empty0 + 8 * slot, phase ^ 1u);
                if (ptx::elect_one()) {
                    ptx::mbar_arrive_expect_tx(raw_full0 + 8 * slot, kRawBytes);
                    // the sample axis is cut into [spectrum][256] (rank 3), so a box never needs a coordinate beyond 2^31
                    const uint32_t dst = base + kOffRaw + slot * kRawBytes;
                    ptx::tma_load_3d(dst, &tmap_raw, raw_full0 + 8 * slot, 0, static_cast<int>(a), m0);
                    ptx::tma_load_3d(dst + kRawBytes / 2, &tmap_raw, raw_full0 + 8 * slot, 128, static_cast<int>(a), m0);
                }
                __syncwarp();
                ++pos;
            }
        }
    } else if (warp == 1) {
        // ===================== MMA issuer (whole warp in uniform control flow, one elected lane issues) =====================
        const uint32_t tb = ptx::uniform(tmem_base);
        uint32_t it = 0;
        for (long long t = first; t < prm.n_tiles; t += step, ++it) {
            const uint32_t buf = it & 1u;
            const uint32_t a_tmem = tb + kTmemA + buf * kTmemABuf;
            ptx::mbar_wait_uniform(a_full0 + 8 * buf, (it >> 1) & 1u);
            ptx::mbar_wait_uniform(re_empty, (it & 1u) ^ 1u);
            ptx::tc_fence_after();
            if (ptx::elect_one()) {
#pragma unroll
                for (int hl = 0; hl < 2; ++hl)
#pragma unroll
                    for (int ks = 0; ks < kFold / 16; ++ks) {
                        // B: K-major SWIZZLE_128B: a k-step is 32 bytes inside the 128-byte row, the second 64-sample chunk
                        // is 128 rows * 128 bytes further; SBO = 8 rows * 128 B.  A: 8 TMEM columns per k-step
                        const uint32_t sb = base + kOffTw + hl * kMatBytes + (ks >> 2) * (kMatBytes / 2) + (ks & 3) * 32;
                        ptx::mma_f16_ts(tb + kTmemRe, a_tmem + 8 * ks, ptx::smem_desc_sw128(sb, 16, 1024), kIdesc, (hl | ks) ? 1u : 0u);
                    }
                // + (-1)^k s[128]: the first k-step of o (o[0] carries s[128]) against the Nyquist sign matrix
                ptx::mma_f16_ts(tb + kTmemRe, a_tmem + 64, ptx::smem_desc_sw128(base + kOffNyq, 16, 1024), kIdesc, 1u);
                ptx::mma_commit(re_full);
            }
            __syncwarp();
            ptx::mbar_wait_uniform(im_empty, (it & 1u) ^ 1u);
            ptx::tc_fence_after();
            if (ptx::elect_one()) {
#pragma unroll
                for (int hl = 0; hl < 2; ++hl)
#pragma unroll
                    for (int ks = 0; ks < kFold / 16; ++ks) {
                        const uint32_t sb = base + kOffTw + (2 + hl) * kMatBytes + (ks >> 2) * (kMatBytes / 2) + (ks & 3) * 32;
                        ptx::mma_f16_ts(tb + kTmemIm, a_tmem + 64 + 8 * ks, ptx::smem_desc_sw128(sb, 16, 1024), kIdesc, (hl | ks) ? 1u : 0u);
                    }
                ptx::mma_commit(im_full);
                ptx::mma_commit(a_empty0 + 8 * buf);         // e / o may be overwritten once these MMAs have read them
            }
            __syncwarp();
        }
    } else if (warp < 2 + kFoldWarps) {
        // ===================== fold + convert: raw int8 -> e, o (fp16) -> the A buffer in tensor memory =====================
        const int quarter = warp & 3;                        // TMEM lanes [32 quarter, +32) = tile rows
        const int jh = (warp - 2) >> 2;                      // sample groups j = 4 jh .. 4 jh + 3 (n = 16 j .. 16 j + 15)
        const int h = quarter >> 1;                          // half tile of this warp's rows
        const int r = (quarter & 1) * 32 + lane;             // row (stream) within the half tile
        const uint32_t lane_addr = tmem_base + (static_cast<uint32_t>(quarter * 32) << 16);
        uint32_t it = 0;
        for (long long t = first; t < prm.n_tiles; t += step, ++it) {
            const uint32_t buf = it & 1u;
            const bool valid = 2 * t + h < prm.n_half;
            const long long pos = 2 * static_cast<long long>(it) + h;
            const int slot = static_cast<int>(pos % kRing);
            // ORDER MATTERS.  The A buffer first: once the MMAs of tile it - 2 have been committed, every fold warp has finished
            // tile it - 2, so every load up to that tile has landed.  Only then is the parity wait on the raw slot sound: the
            // ring is 5 deep and a tile takes 2 slots, so the previous user of this slot is the OTHER half's warps (tile it - 2
            // or it - 3), and TMA loads complete out of order.  Waiting on the slot first, a fast warp could meet the barrier
            // one phase behind (the older load still in flight under DRAM load), which a parity wait reads as "done": stale
            // samples, an extra arrival on raw_empty, and eventually a corrupted barrier (seen as 1 failed launch in 15).
            ptx::mbar_wait_uniform(a_empty0 + 8 * buf, ((it >> 1) & 1u) ^ 1u);   // the MMAs of two tiles ago have read this A buffer
            ptx::tc_fence_after();
            if (valid) ptx::mbar_wait_uniform(raw_full0 + 8 * slot, static_cast<uint32_t>(pos / kRing) & 1u);
            if (valid) {
                const uint32_t raw = base + kOffRaw + slot * kRawBytes;
                const uint32_t a_tmem = lane_addr + kTmemA + buf * kTmemABuf;
                // partner of n = 16 j + i is s[256 - n]: i = 0 -> the byte after the block b (none for n = 0), i >= 1 -> b[16 - i]
                uint32_t nxt = jh ? lds_u32(raw_unit(raw, 1, r, 4)) : 0u;             // s[192] for j = 4
#pragma unroll
                for (int jj = 0; jj < 4; ++jj) {
                    const int j = 4 * jh + jj;
                    const uint4 f = lds_v4(raw_unit(raw, 0, r, j));                    // s[16 j + 0 .. 15]
                    const uint4 b = lds_v4(raw_unit(raw, 1, r, 7 - j));                // s[240 - 16 j + 0 .. 15]
                    const uint32_t q0 = __byte_perm(b.w, nxt, 0x1234), q1 = __byte_perm(b.z, b.w, 0x1234);
                    const uint32_t q2 = __byte_perm(b.y, b.z, 0x1234), q3 = __byte_perm(b.x, b.y, 0x1234);
                    nxt = b.x;                                                          // s[256 - 16 (j + 1)] is its first byte
                    const uint32_t fw[4] = {f.x, f.y, f.z, f.w}, qw[4] = {q0, q1, q2, q3};
                    uint32_t e[8], o[8];
#pragma unroll
                    for (int w = 0; w < 4; ++w) {
                        uint32_t f_lo, f_hi, q_lo, q_hi;
                        bytes_to_half2(fw[w], f_lo, f_hi);
                        bytes_to_half2(qw[w], q_lo, q_hi);
                        e[2 * w] = hadd2(f_lo, q_lo);
                        e[2 * w + 1] = hadd2(f_hi, q_hi);
                        o[2 * w] = hsub2(f_lo, q_lo);
                        o[2 * w + 1] = hsub2(f_hi, q_hi);
                    }
                    if (j == 0) {                            // o[0] (sine zero) carries s[128] for the Nyquist k-step
                        uint32_t s_lo, s_hi;
                        bytes_to_half2(lds_u32(raw_unit(raw, 1, r, 0)), s_lo, s_hi);
                        o[0] = __byte_perm(o[0], s_lo, 0x3254);                       // {low half: s[128], high half: o[1]}
                    }
                    ptx::tmem_st_32x8(a_tmem + 8 * j, e);
                    ptx::tmem_st_32x8(a_tmem + 64 + 8 * j, o);
                }
                ptx::tmem_st_wait();
            }
            ptx::tc_fence_before();
            __syncwarp();
            if (lane == 0) {
                ptx::mbar_arrive(a_full0 + 8 * buf);
                if (valid) ptx::mbar_arrive(raw_empty0 + 8 * slot);
            }
        }
    } else {
        // ===================== epilogue =====================
        const int quarter = warp & 3;                        // TMEM lanes [32 quarter, +32) = tile rows = streams
        const int chalf = (warp - 2 - kFoldWarps) >> 2;      // channels 64 chalf .. + 63
        const int h = quarter >> 1;
        const int r = (quarter & 1) * 32 + lane;
        const uint32_t lane_addr = tmem_base + (static_cast<uint32_t>(quarter * 32) << 16);
        using OutT = typename std::conditional<kInt8, uint16_t, uint32_t>::type;     // one (re, im) pair of one stream
        OutT* out = static_cast<OutT*>(prm.out);
        const uint64_t policy = ptx::policy_evict_first();
        const int pair_id = 2 * h + chalf;                   // the two warps (quarters 2h, 2h + 1) of a half tile and channel half
        const uint32_t xchg = base + kOffRaw + kRawRingI8 * kRawBytes + pair_id * kXchgBytes;     // (kInt8 only)
        uint32_t it = 0;
        for (long long t = first; t < prm.n_tiles; t += step, ++it) {
            const long long hidx = 2 * t + h;
            const bool valid = hidx < prm.n_half;
            const long long a = hidx / n_sb;
            const int m0 = static_cast<int>(hidx - a * n_sb) * kTileStreams;
            OutT* dst = out + (a * kChan + 64 * chalf) * prm.n_stream + m0 + r;         // channel 64 chalf of this stream
            OutT* dst_line = out + (a * kChan + 64 * chalf) * prm.n_stream + m0;        // ... of the half tile's first stream
            const bool row_ok = !kRagged || m0 + r < prm.n_stream;        // this thread's stream exists (ragged last half tile)
            const bool pair_ok = !kRagged || m0 + 2 * lane < prm.n_stream;    // int8 output: the two streams this lane ships (n_stream is even)
            uint32_t rr[32];                                 // Re of this thread's 64 channels as packed pairs
            ptx::mbar_wait_uniform(re_full, it & 1u);
            ptx::tc_fence_after();
#pragma unroll
            for (int part = 0; part < 2; ++part) {
                uint32_t v[32];
                ptx::tmem_ld_32x32(lane_addr + kTmemRe + 64 * chalf + 32 * part, v);
                ptx::tmem_ld_wait();
                if (part == 1) {                             // this warp's part of Re is in registers
                    ptx::tc_fence_before();
                    __syncwarp();
                    if (lane == 0) ptx::mbar_arrive(re_empty);
                }
#pragma unroll
                for (int c = 0; c < 16; ++c)
                    rr[16 * part + c] = pack_pair<kInt8>(__uint_as_float(v[2 * c]), __uint_as_float(v[2 * c + 1]), prm.scale);
            }
            ptx::mbar_wait_uniform(im_full, it & 1u);
            ptx::tc_fence_after();
#pragma unroll
            for (int part = 0; part < 2; ++part) {
                uint32_t v[32];
                ptx::tmem_ld_32x32(lane_addr + kTmemIm + 64 * chalf + 32 * part, v);
                ptx::tmem_ld_wait();
                if (part == 1) {
                    ptx::tc_fence_before();
                    __syncwarp();
                    if (lane == 0) ptx::mbar_arrive(im_empty);
                }
                if (valid) {
                    if constexpr (kInt8) {
                        // this warp's 32 channels x 32 streams of codes into the pair's exchange buffer [channel][64 streams x 2 B]
#pragma unroll
                        for (int c = 0; c < 16; ++c) {
                            const uint32_t ii = pack_pair<kInt8>(__uint_as_float(v[2 * c]), __uint_as_float(v[2 * c + 1]), prm.scale);
                            const uint32_t re2 = rr[16 * part + c];
                            sts_u16(xchg + (2 * c) * 128 + (quarter & 1) * 64 + lane * 2, __byte_perm(re2, ii, 0x0040));
                            sts_u16(xchg + (2 * c + 1) * 128 + (quarter & 1) * 64 + lane * 2, __byte_perm(re2, ii, 0x0051));
                        }
                        pair_sync(1 + pair_id);              // both halves of the 32 rows are in the buffer
                        // each warp ships 16 of the 32 rows as full 128-byte lines (lane = streams 2 lane, 2 lane + 1)
#pragma unroll
                        for (int k = 0; k < 16; ++k) {
                            const int ch = (quarter & 1) * 16 + k;
                            const uint32_t word = lds_u32(xchg + ch * 128 + lane * 4);
                            if (pair_ok)
                                stg_stream(reinterpret_cast<uint32_t*>(dst_line + static_cast<long long>(32 * part + ch) * prm.n_stream) + lane, word, policy);
                        }
                        pair_sync(1 + pair_id);              // the buffer may be overwritten
                    } else {
#pragma unroll
                        for (int c = 0; c < 16; ++c) {
                            const uint32_t ii = pack_pair<kInt8>(__uint_as_float(v[2 * c]), __uint_as_float(v[2 * c + 1]), prm.scale);
                            const uint32_t re2 = rr[16 * part + c];
                            OutT* d0 = dst + static_cast<long long>(32 * part + 2 * c) * prm.n_stream;
                            // (re, im) half2 words of channels 2c and 2c + 1: one 128-byte line per channel and warp
                            // (lane pairs trading words for 8-byte stores of two lines per instruction: no gain, the
                            // write path is bound by lines, not by instructions)
                            if (row_ok) {
                                stg_stream(d0, __byte_perm(re2, ii, 0x5410), policy);
                                stg_stream(d0 + prm.n_stream, __byte_perm(re2, ii, 0x7632), policy);
                            }
                        }
                    }
                }
            }
        }
    }

    ptx::tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        ptx::tc_fence_after();
        ptx::tmem_dealloc(tmem_base, kTmemCols);
    }
}

}  // namespace fengtc
