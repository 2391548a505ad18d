// fengine_tc.cuh -- the F-engine as a dense contraction on tcgen05 tensor cores.
//
// PAPER.md:49-52 (Sec. 2, Eq. 1):  S[k] = sum_{n=0}^{N-1} s[n] exp(-j (2 pi / N) k n),  N = 256, on
// consecutive blocks of every stream's 8-bit REAL samples.  For real input the sum folds onto n = 0 .. 128:
//     e[0] = s[0],  e[n] = s[n] + s[256 - n],  o[n] = s[n] - s[256 - n]      (n = 1 .. 127; integers, exact in fp16)
//     Re S[k] =  sum_{n=0}^{127} e[n] cos(2 pi k n / 256)  +  (-1)^k s[128]
//     Im S[k] = -sum_{n=1}^{127} o[n] sin(2 pi k n / 256)
// i.e. two [128 channels] x [128 samples] matrices applied to the folded samples of every (stream, spectrum): a GEMM
// with M = 128 (channels), K = 128 (folded samples), N = the streams of a tile.  The twiddle matrices are split into
// fp16 hi + lo parts (cos = hi + lo to ~3e-8 absolute), every product e * hi, e * lo is exact in the fp32 accumulator,
// so the result carries only the accumulation round-off: well inside the fp32 bound the parity test allows
// (0.5 ulp of the fp16 output + 2e-6 sum|s|).  Per real sample: 256 tensor MACs instead of ~29 CUDA-core instructions.
//
// One CTA (cta_group::1, 576 threads, persistent over tiles of 64 streams x 1 spectrum):
//   warp 0      TMA: the raw int8 tile [64 streams][256 samples] of every tile into a 4-deep ring
//   warp 1      tcgen05.mma issuer: per tile 32 MMAs (M 128, N 64, K 16): {cos, sin} x {hi, lo} x 8 k-steps into two
//               64-column fp32 accumulators in TMEM (double buffered across tiles).  The A operand -- the four twiddle
//               matrices -- lives in TENSOR MEMORY for the whole kernel (256 columns, written once by warps 2-5 with
//               tcgen05.st), so an MMA reads only its 2 KB of B from shared memory (with A in shared memory the MMAs
//               were shared-memory-bandwidth bound at 2.3x their tensor time, and the 128 KB left no room to double
//               buffer B)
//   warps 2-9   fold + convert: raw int8 -> e, o as fp16 in the K-major SWIZZLE_128B layout the MMA reads (bytes are
//               turned into halves with the 0x6400 | byte trick, no integer-to-float conversion instruction), 2-deep
//   warps 10-17 epilogue (two warps per TMEM lane quarter, 32 streams each): TMEM -> (+ (-1)^k s[128]) -> fp16 (re, im)
//               -> shared-memory transpose -> 128-byte rows of 32 streams per channel, written with 16-byte coalesced
//               stores straight into the X-engine's input layout
// (Round 2, first version: four fold and four epilogue warps, 2-deep raw ring: every role ~80 % busy in a chain of 2-deep
// hand-overs, 2820 clk per tile, 4.56 TB/s.  Eight + eight warps halve the per-tile time of both roles.)
#pragma once
#include <cuda_fp16.h>
#include "ptx.cuh"

namespace fengtc {

constexpr int kFft = 256;
constexpr int kChan = 128;                    // channels kept = MMA M
constexpr int kFold = 128;                    // folded samples = GEMM K
constexpr int kTileStreams = 64;              // streams per tile = MMA N
constexpr int kFoldWarps = 8, kEpiWarps = 8;
constexpr int kThreads = 64 + 32 * (kFoldWarps + kEpiWarps);
constexpr int kRawRing = 4;                   // raw int8 tiles in flight per CTA (covers the DRAM latency)
constexpr int kMatCols = kFold / 2;           // one fp16 twiddle matrix in TMEM: 128 lanes x 64 columns (2 halves each)
constexpr int kRawBytes = kTileStreams * kFft;              // 16 KB
constexpr int kOpBytes = kTileStreams * kFold * 2;          // e or o as fp16: 16 KB (two chunks of 8 KB)
constexpr int kStageRow = 128 + 16;                          // epilogue staging row (32 half2 + pad), bytes
constexpr int kStageWarpBytes = 32 * kStageRow;
// s[128] of a tile travels from the fold warps to the epilogue through this ring.  fold(t) may start once MMA(t - 2) has
// been committed, i.e. once every epilogue warp has RELEASED the accumulator of tile t - 4 -- at which point tile t - 5 is
// finished in every epilogue warp, but tile t - 4 may still be reading its s[128]: the ring must hold >= 5 tiles
constexpr int kS128Ring = 8;
// tensor memory map (columns): two accumulator sets {cos 64, sin 64}, then cos_hi, cos_lo, sin_hi, sin_lo
constexpr int kTmemAcc = 0, kTmemA = 256, kTmemCols = 512;
// shared memory map (offsets from the 1024-byte aligned base)
constexpr int kOffE = 0;                                     // 2 x {e, o}: slot s at s * 2 * kOpBytes
constexpr int kOffO = kOpBytes;
constexpr int kOffRaw = 4 * kOpBytes;                        // kRawRing x 16 KB
constexpr int kOffStage = kOffRaw + kRawRing * kRawBytes;
constexpr int kOffS128 = kOffStage + kEpiWarps * kStageWarpBytes;
constexpr int kOffBar = kOffS128 + kS128Ring * kTileStreams * 4;
constexpr int kSmemBytes = kOffBar + 192 + 1024 /*alignment slack*/;
static_assert(kSmemBytes <= 227 * 1024, "shared memory");

struct Params {
    void* out;               // [n_spectra][128][n_stream] __half2 (re, im)
    const uint4* tw;         // DEVICE: twiddles [cos_hi | cos_lo | -sin_hi | -sin_lo][128 channels][128 samples] fp16
    int n_stream;            // multiple of 64
    long long n_spectra;
    long long n_tiles;       // n_spectra * n_stream / 64
};

// instruction descriptor: D = F32 (1 << 4), A = B = F16, both K-major, M = 128 (8 << 24), N = 64 (8 << 17)
constexpr uint32_t kIdesc = (1u << 4) | (8u << 24) | (static_cast<uint32_t>(kTileStreams >> 3) << 17);

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
__device__ __forceinline__ void sts_v4(uint32_t addr, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
    asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(a), "r"(b), "r"(c), "r"(d) : "memory");
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

__global__ void __launch_bounds__(kThreads, 1)
fengine_tc_kernel(const __grid_constant__ CUtensorMap tmap_raw, const Params prm) {
    extern __shared__ uint8_t smem_raw[];
    const uint32_t base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t bar = base + kOffBar;
    // barriers: a_full, raw_full[4], raw_empty[4], b_full[2], b_empty[2], acc_full[2], acc_empty[2], then the TMEM base word
    const uint32_t a_full = bar, raw_full0 = bar + 8, raw_empty0 = raw_full0 + 8 * kRawRing, b_full0 = raw_empty0 + 8 * kRawRing;
    const uint32_t b_empty0 = b_full0 + 16, acc_full0 = b_empty0 + 16, acc_empty0 = acc_full0 + 16, tmem_slot = acc_empty0 + 16;
    static_assert(8 + 16 * kRawRing + 64 + 4 <= 192, "barrier region");
    uint32_t* tmem_slot_ptr = reinterpret_cast<uint32_t*>(smem_raw + (tmem_slot - ptx::smem_u32(smem_raw)));

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;

    if (threadIdx.x == 0) {
        ptx::prefetch_tensormap(&tmap_raw);
        ptx::mbar_init(a_full, 4);                          // one arrive per uploading warp once its twiddle rows are in TMEM
        for (int k = 0; k < kRawRing; ++k) {
            ptx::mbar_init(raw_full0 + 8 * k, 1);
            ptx::mbar_init(raw_empty0 + 8 * k, kFoldWarps); // one arrive per fold warp
        }
        for (int k = 0; k < 2; ++k) {
            ptx::mbar_init(b_full0 + 8 * k, kFoldWarps);
            ptx::mbar_init(b_empty0 + 8 * k, 1);
            ptx::mbar_init(acc_full0 + 8 * k, 1);
            ptx::mbar_init(acc_empty0 + 8 * k, kEpiWarps);  // one arrive per epilogue warp
        }
        ptx::fence_mbar_init();
    }
    if (warp == 1) {
        ptx::tmem_alloc(tmem_slot, kTmemCols);
        ptx::tmem_relinquish();
    }
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_ptr;

    const int n_sb = prm.n_stream / kTileStreams;           // stream blocks per spectrum: consecutive tiles share a spectrum
    const long long first = blockIdx.x, step = gridDim.x;

    if (warp == 0) {
        // ===================== TMA producer (one elected lane of the converged warp) =====================
        {
            int slot = 0;
            uint32_t phase = 0;
            for (long long t = first; t < prm.n_tiles; t += step) {
                const long long a = t / n_sb;
                const int m0 = static_cast<int>(t - a * n_sb) * kTileStreams;
                ptx::mbar_wait(raw_empty0 + 8 * slot, phase ^ 1u);
                if (ptx::elect_one()) {
                    ptx::mbar_arrive_expect_tx(raw_full0 + 8 * slot, kRawBytes);
                    // the sample axis is cut into [spectrum][256] (rank 3), so a box never needs a coordinate beyond 2^31
                    ptx::tma_load_3d(base + kOffRaw + slot * kRawBytes, &tmap_raw, raw_full0 + 8 * slot, 0, static_cast<int>(a), m0);
                }
                __syncwarp();
                if (++slot == kRawRing) { slot = 0; phase ^= 1u; }
            }
        }
    } else if (warp == 1) {
        // ===================== MMA issuer (whole warp in uniform control flow, one elected lane issues) =====================
        {
            const uint32_t tb = ptx::uniform(tmem_base);
            ptx::mbar_wait(a_full, 0);
            ptx::tc_fence_after();
            uint32_t phase = 0;                              // B slot, accumulator set and their phases advance together
            int slot = 0;
            for (long long t = first; t < prm.n_tiles; t += step) {
                ptx::mbar_wait(b_full0 + 8 * slot, phase);
                ptx::mbar_wait(acc_empty0 + 8 * slot, phase ^ 1u);
                ptx::tc_fence_after();
                if (ptx::elect_one()) {
#pragma unroll
                    for (int part = 0; part < 2; ++part) {       // 0: cos x e -> Re, 1: sin x o -> Im
                        const uint32_t d_tmem = tb + kTmemAcc + slot * 128 + part * 64;
                        const uint32_t sb = base + slot * 2 * kOpBytes + (part ? kOffO : kOffE);
#pragma unroll
                        for (int hl = 0; hl < 2; ++hl) {
                            const uint32_t a_tmem = tb + kTmemA + (2 * part + hl) * kMatCols;
#pragma unroll
                            for (int ks = 0; ks < kFold / 16; ++ks) {
                                // B: K-major SWIZZLE_128B: a k-step is 32 bytes inside the 128-byte row, the second 64-sample
                                // chunk is 64 rows * 128 bytes further; SBO = 8 rows * 128 B.  A: 8 TMEM columns per k-step
                                const uint32_t b_off = (ks >> 2) * (kOpBytes / 2) + (ks & 3) * 32;
                                const uint64_t bdesc = ptx::smem_desc_sw128(sb + b_off, 16, 1024);
                                ptx::mma_f16_ts(d_tmem, a_tmem + 8 * ks, bdesc, kIdesc, (hl | ks) ? 1u : 0u);
                            }
                        }
                    }
                    ptx::mma_commit(b_empty0 + 8 * slot);        // e / o may be overwritten once these MMAs have read them
                    ptx::mma_commit(acc_full0 + 8 * slot);
                }
                __syncwarp();
                if (++slot == 2) { slot = 0; phase ^= 1u; }
            }
        }
    } else if (warp < 2 + kFoldWarps) {
        // ===================== fold + convert: raw int8 -> e, o (fp16, K-major SWIZZLE_128B) =====================
        if (warp < 6) {   // the twiddle matrices into tensor memory, once: row (channel) 32 (warp % 4) + lane of every matrix
            const int krow = (warp & 3) * 32 + lane;
#pragma unroll 1
            for (int m = 0; m < 4; ++m) {
                const uint4* src = prm.tw + (m * kChan + krow) * (kFold * 2 / 16);
#pragma unroll
                for (int half = 0; half < 2; ++half) {
                    uint32_t v[32];
#pragma unroll
                    for (int q = 0; q < 8; ++q) {
                        const uint4 x = __ldg(src + 8 * half + q);
                        v[4 * q] = x.x; v[4 * q + 1] = x.y; v[4 * q + 2] = x.z; v[4 * q + 3] = x.w;
                    }
                    ptx::tmem_st_32x32(tmem_base + (static_cast<uint32_t>((warp & 3) * 32) << 16) + kTmemA + m * kMatCols + 32 * half, v);
                }
            }
            ptx::tmem_st_wait();
            ptx::tc_fence_before();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(a_full);
        }
        const int ct = threadIdx.x - 64;                    // 0 .. 255
        const int j = ct & 7;                                // samples n = 16 j .. 16 j + 15 of the stream
        int slot = 0, rslot = 0;
        uint32_t phase = 0, rphase = 0;                      // B slot / raw slot and their phases
        long long it_tile = 0;
        for (long long t = first; t < prm.n_tiles; t += step, ++it_tile) {
            ptx::mbar_wait(raw_full0 + 8 * rslot, rphase);
            ptx::mbar_wait(b_empty0 + 8 * slot, phase ^ 1u); // the MMAs of two tiles ago have read this e / o slot
            const uint32_t raw = base + kOffRaw + rslot * kRawBytes;
            const uint32_t opb = base + slot * 2 * kOpBytes;
            const uint32_t s128 = base + kOffS128 + static_cast<uint32_t>(it_tile & (kS128Ring - 1)) * (kTileStreams * 4);
#pragma unroll
            for (int rep = 0; rep < kTileStreams / (4 * kFoldWarps); ++rep) {
                const int r = (ct >> 3) + 4 * kFoldWarps * rep;   // stream within the tile
                const uint32_t row = raw + r * kFft;
                const uint4 f = lds_v4(row + 16 * j);                          // s[16 j + 0 .. 15]
                const uint4 b = lds_v4(row + 240 - 16 * j);                    // s[240 - 16 j + 0 .. 15]
                // partner of n = 16 j + i is s[256 - n]: i = 0 -> the byte after the block (none for n = 0), i >= 1 -> b[16 - i]
                const uint32_t nxt = j ? lds_u32(row + 256 - 16 * j) : 0u;
                const uint32_t q0 = __byte_perm(b.w, nxt, 0x1234), q1 = __byte_perm(b.z, b.w, 0x1234);
                const uint32_t q2 = __byte_perm(b.y, b.z, 0x1234), q3 = __byte_perm(b.x, b.y, 0x1234);
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
                // row r of the [64 streams][128 folded samples] operand: chunk j / 4, 16-byte units 2 (j % 4) and + 1
                const uint32_t rowoff = (j >> 2) * (kOpBytes / 2) + (r >> 3) * 1024 + (r & 7) * 128;
                const uint32_t u0 = ((2 * (j & 3)) ^ (r & 7)) * 16, u1 = ((2 * (j & 3) + 1) ^ (r & 7)) * 16;
                sts_v4(opb + kOffE + rowoff + u0, e[0], e[1], e[2], e[3]);
                sts_v4(opb + kOffE + rowoff + u1, e[4], e[5], e[6], e[7]);
                sts_v4(opb + kOffO + rowoff + u0, o[0], o[1], o[2], o[3]);
                sts_v4(opb + kOffO + rowoff + u1, o[4], o[5], o[6], o[7]);
                if (j == 0) {                                // s[128] goes straight to the epilogue
                    const int v = static_cast<int>(static_cast<int8_t>(lds_u32(row + 128) & 0xffu));
                    asm volatile("st.shared.f32 [%0], %1;" ::"r"(s128 + 4 * r), "f"(static_cast<float>(v)) : "memory");
                }
            }
            ptx::fence_proxy_async_smem();                   // generic-proxy writes -> visible to the tensor core
            __syncwarp();
            if (lane == 0) {
                ptx::mbar_arrive(b_full0 + 8 * slot);
                ptx::mbar_arrive(raw_empty0 + 8 * rslot);
            }
            if (++slot == 2) { slot = 0; phase ^= 1u; }
            if (++rslot == kRawRing) { rslot = 0; rphase ^= 1u; }
        }
    } else {
        // ===================== epilogue =====================
        const int quarter = warp & 3;                        // TMEM lanes [32 quarter, +32) = channels
        const int k = quarter * 32 + lane;                   // this thread's channel
        const float sgn = (k & 1) ? -1.0f : 1.0f;
        const int hh = (warp - 2 - kFoldWarps) >> 2;        // this warp's 32 streams of the tile
        const uint32_t stage = base + kOffStage + (warp - 2 - kFoldWarps) * kStageWarpBytes;
        __half2* out = static_cast<__half2*>(prm.out);
        uint32_t acc_phase = 0;
        int acc = 0;
        long long it_tile = 0;
        for (long long t = first; t < prm.n_tiles; t += step, ++it_tile) {
            const long long a = t / n_sb;
            const int m0 = static_cast<int>(t - a * n_sb) * kTileStreams;
            const uint32_t s128 = base + kOffS128 + static_cast<uint32_t>(it_tile & (kS128Ring - 1)) * (kTileStreams * 4);
            ptx::mbar_wait(acc_full0 + 8 * acc, acc_phase);
            ptx::tc_fence_after();
            const uint32_t taddr = tmem_base + (static_cast<uint32_t>(quarter * 32) << 16) + kTmemAcc + acc * 128;
            {
                uint32_t re[32], im[32];
                ptx::tmem_ld_32x32(taddr + 32 * hh, re);
                ptx::tmem_ld_32x32(taddr + 64 + 32 * hh, im);
                ptx::tmem_ld_wait();
                ptx::tc_fence_before();                      // this warp's part is in registers
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive(acc_empty0 + 8 * acc);
                uint32_t h[32];
#pragma unroll
                for (int c4 = 0; c4 < 8; ++c4) {
                    const uint4 sv = lds_v4(s128 + (32 * hh + 4 * c4) * 4);          // broadcast: s[128] of four streams
                    const float s4[4] = {__uint_as_float(sv.x), __uint_as_float(sv.y), __uint_as_float(sv.z), __uint_as_float(sv.w)};
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        const int c = 4 * c4 + q;
                        const __half2 v = __floats2half2_rn(fmaf(sgn, s4[q], __uint_as_float(re[c])), __uint_as_float(im[c]));
                        h[c] = *reinterpret_cast<const uint32_t*>(&v);
                    }
                }
                // transpose through shared memory: row = channel (this lane), 32 streams x 4 bytes
                __syncwarp();                                // the previous tile has been read out of the staging rows
#pragma unroll
                for (int c4 = 0; c4 < 8; ++c4)
                    sts_v4(stage + lane * kStageRow + 16 * c4, h[4 * c4], h[4 * c4 + 1], h[4 * c4 + 2], h[4 * c4 + 3]);
                __syncwarp();
                // 8 lanes cover one 128-byte output row, 4 rows per instruction
#pragma unroll
                for (int p = 0; p < 8; ++p) {
                    const int rowl = 4 * p + (lane >> 3);
                    const uint4 v = lds_v4(stage + rowl * kStageRow + 16 * (lane & 7));
                    __half2* dst = out + ((a * kChan + quarter * 32 + rowl) * prm.n_stream + m0 + 32 * hh + 4 * (lane & 7));
                    *reinterpret_cast<uint4*>(dst) = v;
                }
            }
            if (++acc == 2) { acc = 0; acc_phase ^= 1u; }
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
