// fengine.cuh -- the F-engine in front of the X-engine.
//
// PAPER.md:49-52 (Sec. 2, Eq. 1):  S[k] = sum_{n=0}^{N-1} s[n] exp(-j (2 pi / N) k n),  N = 256,
// applied to consecutive blocks of every stream's 8-bit real samples.  Output: the N/2 = 128
// non-redundant channels k = 0..127 as complex fp16, written DIRECTLY in the X-engine's input layout
// x[spectrum a][channel k][stream m] -- so no corner turn exists between the two engines.
//
// Two real streams per complex transform: z[n] = s_m[n] + j s_{m+1}[n] (the two polarisations of one station when
// n_pol = 2), Z = DFT256(z), then S_m[k] = (Z[k] + conj(Z[N-k])) / 2 and S_{m+1}[k] = (Z[k] - conj(Z[N-k])) / (2j).
// DFT256 = 16 x 16 (Cooley-Tukey): 16 threads per transform, each computes a 16-point DFT in registers
// (radix 4 x 4) per pass, with one shared-memory exchange between the passes; the pass-A twiddles live in registers and
// the two-stream split pairs Z[k] with Z[N-k] by shuffles.  fp32 arithmetic, fp16 (RN) output.
//
// One block = 32 streams (16 transforms x 16 threads) x 8 consecutive spectra: the 16 threads of a transform read each
// 16-byte run of samples together (one byte each, already in pass-A order), stores are 128-byte rows along the stream
// axis (32 streams x 4 bytes) for each channel.
#pragma once
#include <cuda_fp16.h>
#include <cstdint>

namespace feng {

constexpr int kFft = 256;
constexpr int kChan = kFft / 2;          // channels kept
constexpr int kThreads = 256;
constexpr int kStreamsPerBlock = 32;
constexpr int kPitch = kFft + 16;        // float2 per transform buffer: index n + n / 16 (bank spread)
constexpr int kSpectraPerBlock = 8;      // consecutive spectra per block (amortises the twiddle table and the launch)

struct Params {
    const int8_t* in;        // [n_stream][n_spectra * 256]
    void* out;               // [n_spectra][128][n_stream] (re, im): __half2 (cf16) or char2 (ci8)
    int n_stream;
    long long n_spectra;
    float scale;             // ci8 output only: code = clip(rint(S * scale), -127, 127)
};

// output element: complex fp16 (one rounding to nearest) or requantised complex int8
template <bool kInt8> struct Out;
template <> struct Out<false> {
    using T = __half2;
    static __device__ __forceinline__ T cvt(float re, float im, float) { return __floats2half2_rn(re, im); }
};
template <> struct Out<true> {
    using T = char2;
    static __device__ __forceinline__ T cvt(float re, float im, float scale) {
        const int a = max(-127, min(127, __float2int_rn(re * scale)));      // rint, ties to even; -128 is never produced
        const int b = max(-127, min(127, __float2int_rn(im * scale)));
        return make_char2(static_cast<signed char>(a), static_cast<signed char>(b));
    }
};

__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
    return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ float2 mulmj(float2 a) { return make_float2(a.y, -a.x); }     // a * (-j)

// forward 4-point DFT in place: X[k] = sum_n x[n] exp(-j 2 pi k n / 4)
__device__ __forceinline__ void dft4(float2& x0, float2& x1, float2& x2, float2& x3) {
    const float2 s02 = cadd(x0, x2), d02 = csub(x0, x2);
    const float2 s13 = cadd(x1, x3), d13 = mulmj(csub(x1, x3));      // -j (x1 - x3)
    x0 = cadd(s02, s13);
    x1 = cadd(d02, d13);
    x2 = csub(s02, s13);
    x3 = csub(d02, d13);
}

// forward 16-point DFT: in v[n], out v[k] (natural order).  n = 4a + b, k = c + 4d:
//   X[c + 4d] = sum_b W4^{bd} ( W16^{bc} sum_a x[4a + b] W4^{ac} )
__device__ __forceinline__ void dft16(float2 (&v)[16]) {
    // step 1: for each b, DFT4 over a of x[4a + b]  ->  y_b[c] stored at v[4c + b]
#pragma unroll
    for (int b = 0; b < 4; ++b) dft4(v[b], v[4 + b], v[8 + b], v[12 + b]);
    // step 2: twiddles W16^{bc} = exp(-j pi b c / 8)
    const float c1 = 0.92387953251128674f, s1 = 0.38268343236508977f, r2 = 0.70710678118654752f;
    const float2 w1 = make_float2(c1, -s1), w2 = make_float2(r2, -r2), w3 = make_float2(s1, -c1);
    const float2 w6 = make_float2(-r2, -r2), w9 = make_float2(-c1, s1);
    v[4 * 1 + 1] = cmul(v[4 * 1 + 1], w1);
    v[4 * 1 + 2] = cmul(v[4 * 1 + 2], w2);
    v[4 * 1 + 3] = cmul(v[4 * 1 + 3], w3);
    v[4 * 2 + 1] = cmul(v[4 * 2 + 1], w2);
    v[4 * 2 + 2] = mulmj(v[4 * 2 + 2]);                  // W16^4 = -j
    v[4 * 2 + 3] = cmul(v[4 * 2 + 3], w6);
    v[4 * 3 + 1] = cmul(v[4 * 3 + 1], w3);
    v[4 * 3 + 2] = cmul(v[4 * 3 + 2], w6);
    v[4 * 3 + 3] = cmul(v[4 * 3 + 3], w9);
    // step 3: for each c, DFT4 over b  ->  X[c + 4d] lands at v[4c + d]
#pragma unroll
    for (int c = 0; c < 4; ++c) dft4(v[4 * c], v[4 * c + 1], v[4 * c + 2], v[4 * c + 3]);
    // reorder v[4c + d] -> natural v[c + 4d] (a 4 x 4 transpose of register names; free after unrolling)
#pragma unroll
    for (int c = 0; c < 4; ++c)
#pragma unroll
        for (int d = c + 1; d < 4; ++d) {
            const float2 t = v[4 * c + d];
            v[4 * c + d] = v[4 * d + c];
            v[4 * d + c] = t;
        }
}

template <bool kInt8>
__global__ void __launch_bounds__(kThreads) fengine_kernel(const Params prm) {
    using OutT = typename Out<kInt8>::T;
    __shared__ float2 buf[kThreads / 16][kPitch];                 // one 256-point complex buffer per transform
    // output staging [k][stream in block], aliased onto buf once every transform has been read back into registers
    OutT (*ost)[kStreamsPerBlock + 1] = reinterpret_cast<OutT (*)[kStreamsPerBlock + 1]>(&buf[0][0]);
    static_assert(sizeof(OutT) * kChan * (kStreamsPerBlock + 1) <= sizeof(float2) * (kThreads / 16) * kPitch, "staging fits");

    const int tid = threadIdx.x;
    const int g = tid >> 4;              // transform within the block (stream pair)
    const int c = tid & 15;              // thread within the transform
    // blocks that run together cover ALL streams of the same spectra, so the 128-byte output rows of one (a, k) meet in L2
    const unsigned n_sb = (prm.n_stream + kStreamsPerBlock - 1) / kStreamsPerBlock;
    const unsigned ab = blockIdx.x / n_sb;
    const int m0 = static_cast<int>(blockIdx.x % n_sb) * kStreamsPerBlock;
    const int m = m0 + 2 * g;            // streams m (real part) and m + 1 (imaginary part)

    // pass-A twiddles W256^{n2 k1} = exp(-j 2 pi c k1 / 256) of this thread (n2 = c), kept in registers for all spectra
    float2 twr[16];
#pragma unroll
    for (int k1 = 0; k1 < 16; ++k1) {
        float sn, cs;
        sincospif(-static_cast<float>(c * k1) / 128.0f, &sn, &cs);
        twr[k1] = make_float2(cs, sn);
    }

    const long long row = prm.n_spectra * kFft;
    float2* z = buf[g];
    const long long a_end = (ab + 1ll) * kSpectraPerBlock < prm.n_spectra ? (ab + 1ll) * kSpectraPerBlock : prm.n_spectra;
    for (long long a = static_cast<long long>(ab) * kSpectraPerBlock; a < a_end; ++a) {
    // ---- pass A operands straight from global memory: n = 16 n1 + n2, this thread is n2 = c and takes the 16 samples
    //      n1 = 0..15 (stride 16 bytes) of both streams; the 16 threads of a transform cover each 16-byte run together,
    //      z[n] = s_m[n] + j s_{m+1}[n] ----
    float2 v[16];
    {
        const uint8_t* pa = reinterpret_cast<const uint8_t*>(prm.in) + m * row + a * kFft + c;
        const uint8_t* pb = pa + row;
        const bool oka = m < prm.n_stream, okb = m + 1 < prm.n_stream;
        // int8 -> fp32 on the ALU pipe: the byte b (two's complement of x) gives b ^ 0x80 = x + 128 in [0, 255]; placed in
        // the mantissa of 2^23 it reads as the float 2^23 + x + 128 exactly (an I2F would run on the quarter-rate XU pipe)
        auto cvt = [](uint32_t b) { return __uint_as_float(0x4B000000u | (b ^ 0x80u)) - 8388736.0f; };
#pragma unroll
        for (int n1 = 0; n1 < 16; ++n1)
            v[n1] = make_float2(oka ? cvt(pa[16 * n1]) : 0.0f, okb ? cvt(pb[16 * n1]) : 0.0f);
    }
    dft16(v);
    __syncwarp();                                                 // the 16 threads of a transform share a warp
#pragma unroll
    for (int k1 = 0; k1 < 16; ++k1) {
        const float2 y = cmul(v[k1], twr[k1]);
        z[16 * k1 + c + k1] = y;                                  // [k1][n2]
    }
    __syncwarp();

    // ---- pass B: this thread is k1 = c: DFT16 over n2  ->  Z[k1 + 16 k2] ----
#pragma unroll
    for (int n2 = 0; n2 < 16; ++n2) v[n2] = z[16 * c + n2 + c];
    dft16(v);                                                     // v[k2] = Z[c + 16 k2]

    // ---- split the two real streams: Z[N - k] for k = c + 16 i sits in thread (16 - c) mod 16 as v[15 - i]
    //      (thread 0: its own v[(16 - i) mod 16]); one shuffle pair inside the 16-lane group, no shared memory ----
    OutT h0[kChan / 16], h1[kChan / 16];
    const int partner = (16 - c) & 15;
#pragma unroll
    for (int i = 0; i < kChan / 16; ++i) {
        const float2 p = v[i];                                    // Z[k], k = c + 16 i in 0 .. 127
        float2 q = make_float2(__shfl_sync(0xffffffffu, v[15 - i].x, partner, 16), __shfl_sync(0xffffffffu, v[15 - i].y, partner, 16));
        if (c == 0) q = v[(16 - i) & 15];
        // S_m = (Z[k] + conj(Z[N-k])) / 2 ;  S_{m+1} = (Z[k] - conj(Z[N-k])) / (2j)
        h0[i] = Out<kInt8>::cvt(0.5f * (p.x + q.x), 0.5f * (p.y - q.y), prm.scale);
        h1[i] = Out<kInt8>::cvt(0.5f * (p.y + q.y), 0.5f * (q.x - p.x), prm.scale);
    }
    __syncthreads();                                              // every z[] has been consumed: reuse the memory
#pragma unroll
    for (int i = 0; i < kChan / 16; ++i) {
        ost[c + 16 * i][2 * g] = h0[i];
        ost[c + 16 * i][2 * g + 1] = h1[i];
    }
    __syncthreads();

    // ---- coalesced stores: for every channel k one 128-byte row of 32 streams ----
    const int col = tid & 31;
    if (m0 + col < prm.n_stream) {
#pragma unroll 4
        for (int k = tid >> 5; k < kChan; k += kThreads / 32)
            static_cast<OutT*>(prm.out)[(a * kChan + k) * prm.n_stream + m0 + col] = ost[k][col];
    }
    __syncthreads();                                              // staging (aliased onto buf) is free again
    }   // spectra of this block
}

}  // namespace feng
