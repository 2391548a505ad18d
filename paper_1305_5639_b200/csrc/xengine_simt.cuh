// xengine_simt.cuh -- plain CUDA-core X-engine for geometries TMA cannot address (input row pitch
// C*N*P*sample_bytes not a multiple of 16 bytes).  One thread per stored visibility, Eq. 2
// evaluated term by term.  Not a performance path.
#pragma once
#include <cuda_fp16.h>
#include <cstdint>

namespace xsimt {

struct Params {
    const void* in;
    void* out;
    int n_station, n_pol, n_chan, n_time;
    long long n_baseline;
    long long n_vis;     // n_chan * n_baseline * n_pol * n_pol
    int accumulate;
    // rectangular cross-only mode: second stream from in_b ([T][C][n_station_b][P]); n_baseline is then
    // n_station * n_station_b and visibilities are ordered [c][i][j][p][q].  n_station_b == 0: packed triangle of `in`.
    const void* in_b;
    int n_station_b;
    // channel window: n_chan channels starting at channel chan0 of inputs laid out for n_chan_total channels, written to
    // the output slabs chan0_out ..
    int chan0, n_chan_total, chan0_out;
};

__device__ __forceinline__ void decode_baseline(long long b, int& i, int& j) {
    // largest i with i(i+1)/2 <= b
    long long r = static_cast<long long>((sqrt(8.0 * static_cast<double>(b) + 1.0) - 1.0) * 0.5);
    while (r * (r + 1) / 2 > b) --r;
    while ((r + 1) * (r + 2) / 2 <= b) ++r;
    i = static_cast<int>(r);
    j = static_cast<int>(b - r * (r + 1) / 2);
}

template <bool kFloat>
__global__ void xengine_simt_kernel(const Params prm) {
    const int P = prm.n_pol, N = prm.n_station, C = prm.n_chan_total;
    const long long v_out0 = static_cast<long long>(prm.chan0_out) * prm.n_baseline * P * P;    // first word of the window
    for (long long w = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x; w < prm.n_vis;
         w += static_cast<long long>(gridDim.x) * blockDim.x) {
        const long long v = v_out0 + w;                                                         // output word
        const int q = static_cast<int>(w % P);
        const int p = static_cast<int>((w / P) % P);
        const long long cb = w / (P * P);
        const long long b = cb % prm.n_baseline;
        const int c = prm.chan0 + static_cast<int>(cb / prm.n_baseline);                        // input channel
        int i, j;
        const bool rect = prm.n_station_b > 0;
        if (rect) {
            i = static_cast<int>(b / prm.n_station_b);
            j = static_cast<int>(b % prm.n_station_b);
        } else {
            decode_baseline(b, i, j);
        }
        const int Nb = rect ? prm.n_station_b : N;
        const long long pitch = static_cast<long long>(C) * N * P;          // samples per time step of the first stream
        const long long pitch_b = static_cast<long long>(C) * Nb * P;
        const long long ia = (static_cast<long long>(c) * N + i) * P + p;
        const long long ib = (static_cast<long long>(c) * Nb + j) * P + q;
        if constexpr (kFloat) {
            const __half2* x = static_cast<const __half2*>(prm.in);
            const __half2* xb = rect ? static_cast<const __half2*>(prm.in_b) : x;
            double re = 0.0, im = 0.0;
            for (int t = 0; t < prm.n_time; ++t) {
                const float2 a = __half22float2(x[t * pitch + ia]);
                const float2 bb = __half22float2(xb[t * pitch_b + ib]);
                re += static_cast<double>(a.x) * bb.x + static_cast<double>(a.y) * bb.y;
                im += static_cast<double>(a.x) * bb.y - static_cast<double>(a.y) * bb.x;
            }
            float2* o = static_cast<float2*>(prm.out) + v;
            float2 r = make_float2(static_cast<float>(re), static_cast<float>(im));
            if (prm.accumulate) { r.x += o->x; r.y += o->y; }
            *o = r;
        } else {
            const char2* x = static_cast<const char2*>(prm.in);
            const char2* xb = rect ? static_cast<const char2*>(prm.in_b) : x;
            int re = 0, im = 0;
            for (int t = 0; t < prm.n_time; ++t) {
                const char2 a = x[t * pitch + ia];
                const char2 bb = xb[t * pitch_b + ib];
                re += a.x * bb.x + a.y * bb.y;
                im += a.x * bb.y - a.y * bb.x;
            }
            int2* o = static_cast<int2*>(prm.out) + v;
            int2 r = make_int2(re, im);
            if (prm.accumulate) { r.x += o->x; r.y += o->y; }
            *o = r;
        }
    }
}

}  // namespace xsimt
