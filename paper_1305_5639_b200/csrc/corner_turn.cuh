// corner_turn.cuh -- pre-X-engine corner turn: [time][chan][station][pol] -> channel-major, time-inner.
//
// Flattening cm = c*M + m (m = s*P + p) makes it one 2-D transpose of complex samples,
//     ws    [cm][t] = in[t][cm]
//     ws_rot[cm][t] = (im, -re) of in[t][cm]        (second plane: feeds the imaginary part)
// with the time axis zero-padded to Tp.  Pure data movement (the B200 analogue of the paper's
// "indexing ... for optimizing the GPU memory access"): 128-bit coalesced loads
// along cm, a shared-memory transpose in 32-bit words, 128-bit coalesced stores along t.
//
// One block = one [64 samples of cm] x [32 output words of t] patch.  A 32-bit output word is two
// consecutive time samples of one stream for ci8 (2-byte samples) or one sample for cf16 (4 bytes).
#pragma once
#include <cstdint>

namespace cturn {

constexpr int kThreads = 256;
constexpr int kTileCm = 64;          // streams per tile
constexpr int kTileWords = 32;       // output words along t per tile: 64 samples (ci8) / 32 samples (cf16)
constexpr int kPitch = 33;           // smem row pitch in words

struct Params {
    const void* in;
    void* ws;            // plane 0
    void* ws_rot;        // plane 1 (nullptr: not written)
    long long n_cm;      // C * M
    int n_time;          // T
    int n_time_pad;      // Tp (multiple of 64)
};

__device__ __forceinline__ uint64_t policy_evict_first() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ void stg_stream(void* p, const uint4& v, uint64_t policy) {
    // written once, read by a later kernel: keep it out of L1, let L2 write it back early
    asm volatile("st.global.L1::no_allocate.L2::cache_hint.v4.u32 [%0], {%1, %2, %3, %4}, %5;" ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z),
                 "r"(v.w), "l"(policy)
                 : "memory");
}
__device__ __forceinline__ uint4 ldg_stream(const uint4* p, uint64_t policy) {
    uint4 r;
    // read once: no L1 allocation, first in line for L2 eviction
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.v4.u32 {%0, %1, %2, %3}, [%4], %5;"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
                 : "l"(p), "l"(policy));
    return r;
}

// (re, im) -> (im, -re) on every complex sample packed in a 32-bit word.
template <int kSampleBytes> __device__ __forceinline__ uint32_t rotate_word(uint32_t w) {
    if constexpr (kSampleBytes == 2) {
        const uint32_t sw = __byte_perm(w, 0, 0x2301);          // [im0, re0, im1, re1]
        const uint32_t ng = __vnegss4(sw);                       // bytewise negate, saturating: -(-128) -> 127
        return (sw & 0x00ff00ffu) | (ng & 0xff00ff00u);          // negate the (new) imaginary bytes
    } else {
        return __byte_perm(w, 0, 0x1032) ^ 0x80000000u;          // [im, re] halves, flip sign of the upper
    }
}

template <int kSampleBytes>
__global__ void __launch_bounds__(kThreads)
corner_turn_kernel(const Params prm) {
    __shared__ uint32_t tile[kTileCm * kPitch];

    const long long cm0 = static_cast<long long>(blockIdx.x) * kTileCm;
    const int tid = threadIdx.x;
    const long long in_pitch = prm.n_cm * kSampleBytes;          // bytes per time step
    const uint8_t* in = static_cast<const uint8_t*>(prm.in);
    const uint64_t policy = policy_evict_first();

    if constexpr (kSampleBytes == 2) {
        // 64 t x 64 cm patch.  Thread (tp, chunk): rows 2tp, 2tp+1; streams chunk*8 .. +7 (16 bytes each).
        const int t0 = blockIdx.y * 64;
        const int tp = tid >> 3, chunk = tid & 7;
        const long long cm = cm0 + chunk * 8;
        uint4 a = make_uint4(0, 0, 0, 0), b = make_uint4(0, 0, 0, 0);
        if (cm < prm.n_cm) {
            const int ta = t0 + 2 * tp;
            if (ta < prm.n_time) a = ldg_stream(reinterpret_cast<const uint4*>(in + ta * in_pitch + cm * 2), policy);
            if (ta + 1 < prm.n_time) b = ldg_stream(reinterpret_cast<const uint4*>(in + (ta + 1) * in_pitch + cm * 2), policy);
        }
        const uint32_t aw[4] = {a.x, a.y, a.z, a.w}, bw[4] = {b.x, b.y, b.z, b.w};
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            // aw[k] = samples (cm+2k, cm+2k+1) at time 2tp; bw[k] the same streams at time 2tp+1
            tile[(chunk * 8 + 2 * k) * kPitch + tp] = __byte_perm(aw[k], bw[k], 0x5410);      // low halves
            tile[(chunk * 8 + 2 * k + 1) * kPitch + tp] = __byte_perm(aw[k], bw[k], 0x7632);  // high halves
        }
    } else {
        // 32 t x 64 cm patch.  Thread (trow, chunk): streams chunk*4 .. +3 (16 bytes); two passes of 16 rows.
        const int t0 = blockIdx.y * 32;
        const int trow = tid >> 4, chunk = tid & 15;
        const long long cm = cm0 + chunk * 4;
#pragma unroll
        for (int pass = 0; pass < 2; ++pass) {
            const int tl = trow + 16 * pass;
            uint4 a = make_uint4(0, 0, 0, 0);
            if (cm < prm.n_cm && t0 + tl < prm.n_time)
                a = ldg_stream(reinterpret_cast<const uint4*>(in + (t0 + tl) * in_pitch + cm * 4), policy);
            tile[(chunk * 4 + 0) * kPitch + tl] = a.x;
            tile[(chunk * 4 + 1) * kPitch + tl] = a.y;
            tile[(chunk * 4 + 2) * kPitch + tl] = a.z;
            tile[(chunk * 4 + 3) * kPitch + tl] = a.w;
        }
    }
    __syncthreads();

    // Output: thread (row, tg) writes 16 bytes = words 4tg .. 4tg+3 of stream row; 8 threads cover the
    // 128-byte row segment; two passes of 32 streams.
    const long long out_pitch = static_cast<long long>(prm.n_time_pad) * kSampleBytes;   // bytes per stream row
    const long long seg = static_cast<long long>(blockIdx.y) * 128;                     // byte offset of this patch
    uint8_t* ws = static_cast<uint8_t*>(prm.ws);
    uint8_t* wr = static_cast<uint8_t*>(prm.ws_rot);
    const int tg = tid & 7;
#pragma unroll
    for (int pass = 0; pass < 2; ++pass) {
        const int row = (tid >> 3) + 32 * pass;
        if (cm0 + row < prm.n_cm) {
            const uint32_t* src = tile + row * kPitch + 4 * tg;
            const uint4 v = make_uint4(src[0], src[1], src[2], src[3]);
            const long long off = (cm0 + row) * out_pitch + seg + 16 * tg;
            stg_stream(ws + off, v, policy);
            if (wr != nullptr) {
                const uint4 r = make_uint4(rotate_word<kSampleBytes>(v.x), rotate_word<kSampleBytes>(v.y),
                                           rotate_word<kSampleBytes>(v.z), rotate_word<kSampleBytes>(v.w));
                stg_stream(wr + off, r, policy);
            }
        }
    }
}

}  // namespace cturn
