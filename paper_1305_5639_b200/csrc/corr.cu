// corr.cu -- libcorr.so: C ABI (include/corr.h), plan / tile schedule / launch logic.
// The device code lives in xengine_tc.cuh (tcgen05 HERK + packed writer + accumulate),
// corner_turn.cuh (piece a) and xengine_simt.cuh (geometries TMA cannot address).
#include "../../include/corr.h"

#include <cuda.h>
#include <cuda_runtime.h>

#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cmath>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "corner_turn.cuh"
#include "fengine.cuh"
#include "fengine_tc.cuh"
#include "xengine_simt.cuh"
#include "xengine_tc.cuh"
#include "xengine_pair.cuh"

namespace {

constexpr long long kMaxIntegrationCi8 = 65535;   // 2 * 128^2 * T_total <= 2^31 - 1
constexpr unsigned kSchedRing = 256;              // launches in flight on different streams never share a feed counter
constexpr int kMapCache = 16;                     // encoded tensor maps kept per handle (config 4 cycles four inputs)
constexpr int kHostWindows = 8;                   // corr_xengine_host: channel windows in flight through the copy pipeline

thread_local char g_create_error[512] = "";

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// What one launch addresses: `n_chan` channels starting at `chan0_in` of an input laid out for `c_total_in` channels
// ([n_dump][n_time][c_total_in][M]), written to slabs `chan0_out`.. of an output laid out for `c_total_out` channels.
struct View {
    int n_time;            // samples per integration
    int n_chan;
    int c_total_in, chan0_in;
    int c_total_out, chan0_out;
};

struct MapKey {
    const void* ptr;
    int streams;           // M of the group the map addresses
    int c_total, n_time, n_dump, box_rows;
    bool operator==(const MapKey& o) const {
        return ptr == o.ptr && streams == o.streams && c_total == o.c_total && n_time == o.n_time && n_dump == o.n_dump &&
               box_rows == o.box_rows;
    }
};

}  // namespace

struct corr_plan {
    int N, P, C, T, dtype;
    int C_total, chan0;    // channel window [chan0, chan0 + C) of buffers laid out for C_total channels (whole band: 0, C)
    int M;                 // N * P
    int Nb, Mb;            // rectangular cross-only plan (corr_create_cross): stations / streams of group B; 0 = HERK
    long long B;           // N (N + 1) / 2, or N * Nb for a cross plan
    int sample_bytes;      // 2 (ci8) or 4 (cf16)
    int device;
    int sm_count;
    bool tma_ok;           // one channel's row of components (2*M*elt bytes) is a multiple of 16 bytes, so every
                           // TMA box start (c*2M + tile offset) is 16-byte aligned
    long long t_total;     // samples integrated since the last accumulate == 0 call
    int last_launches;

    int kernel;            // requested CORR_KERNEL_*
    std::vector<xtc::TileDesc> h_tiles;
    xtc::TileDesc* d_tiles;
    std::vector<xtc::PairTile> h_pair_tiles;
    xtc::PairTile* d_pair_tiles;
    unsigned int* d_sched;                     // ring of tile-feed counters, one per launch (kSchedRing)
    unsigned int sched_seq;
    int max_clusters;                          // co-resident CTA pairs (cudaOccupancyMaxActiveClusters)
    EncodeTiledFn encode;

    // encoded tensor maps, least recently used replaced
    MapKey map_key[kMapCache];
    CUtensorMap map_val[kMapCache];
    unsigned long long map_used[kMapCache];
    unsigned long long map_clock;

    // corner-turn feed
    int Tp;                // padded time extent of the workspace

    // corr_xengine_host: device staging (two input windows, the running output) and the copy pipeline
    void* d_in_stage[2];
    void* d_out_stage;
    bool host_sum_valid;   // d_out_stage holds a complete integration (false after a failed corr_xengine_host call)
    cudaStream_t st_h2d, st_run, st_d2h;
    cudaEvent_t ev_h2d[2], ev_run[2];

    char err[512];
};

namespace {

int fail(corr_plan* h, int code, const char* fmt, ...) {
    char* dst = h ? h->err : g_create_error;
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(dst, 512, fmt, ap);
    va_end(ap);
    return code;
}

int fail_cuda(corr_plan* h, cudaError_t e, const char* what) {
    return fail(h, CORR_ECUDA, "%s: %s", what, cudaGetErrorString(e));
}

EncodeTiledFn get_encode_fn() {
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    const cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
    if (e != cudaSuccess || qres != cudaDriverEntryPointSuccess) return nullptr;
    return reinterpret_cast<EncodeTiledFn>(fn);
}

// Tensor-core F-engine (fengine_tc.cuh): per-device twiddle table [cos_hi | cos_lo | -sin_hi | -sin_lo | nyquist], each
// [128 channels][128 folded samples] fp16 (nyquist: (-1)^k in sample slot 0, zero elsewhere); built on first use and kept
// (160 KB per device) until the process exits: freeing it from a static destructor would call into a CUDA runtime that may
// already have shut down.
struct FengTcState {
    bool tried = false, ok = false;
    void* d_tw = nullptr;
    EncodeTiledFn encode = nullptr;
    int sm_count = 0;
};
std::mutex g_feng_mutex;
FengTcState g_feng[64];

FengTcState* fengine_tc_state() {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return nullptr;
    std::lock_guard<std::mutex> lock(g_feng_mutex);
    FengTcState& st = g_feng[dev];
    if (st.tried) return st.ok ? &st : nullptr;
    // `tried` is set only on a DEFINITIVE answer (wrong architecture, no tensor-map encoder, or success): a transient
    // failure of the allocation or the copy below is retried by the next call instead of disabling the kernel for good.
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, dev) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    if (prop.major != 10 || prop.minor != 0) { st.tried = true; return nullptr; }
    st.sm_count = prop.multiProcessorCount;
    st.encode = get_encode_fn();
    if (!st.encode) { st.tried = true; return nullptr; }
    // hi = fp16(w), lo = fp16(w - hi): w = hi + lo to ~3e-8 absolute (lo may be subnormal)
    std::vector<__half> tw(fengtc::kNumMats * fengtc::kChan * fengtc::kFold, __float2half_rn(0.0f));
    const double two_pi = 6.283185307179586476925286766559;
    for (int k = 0; k < fengtc::kChan; ++k)
        for (int n = 0; n < fengtc::kFold; ++n) {
            const int kn = (k * n) % fengtc::kFft;                       // exact angle reduction in integers
            const double c = std::cos(two_pi * kn / fengtc::kFft), sn = -std::sin(two_pi * kn / fengtc::kFft);
            const double w[2] = {c, sn};
            for (int part = 0; part < 2; ++part) {
                const __half hi = __float2half_rn(static_cast<float>(w[part]));
                const __half lo = __float2half_rn(static_cast<float>(w[part] - static_cast<double>(__half2float(hi))));
                tw[((2 * part + 0) * fengtc::kChan + k) * fengtc::kFold + n] = hi;
                tw[((2 * part + 1) * fengtc::kChan + k) * fengtc::kFold + n] = lo;
            }
        }
    for (int k = 0; k < fengtc::kChan; ++k) tw[(4 * fengtc::kChan + k) * fengtc::kFold] = __float2half_rn((k & 1) ? -1.0f : 1.0f);
    void* d_tw = nullptr;
    if (cudaMalloc(&d_tw, tw.size() * sizeof(__half)) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    if (cudaMemcpy(d_tw, tw.data(), tw.size() * sizeof(__half), cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaFuncSetAttribute(fengtc::fengine_tc_kernel<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, fengtc::kSmemBytes) != cudaSuccess ||
        cudaFuncSetAttribute(fengtc::fengine_tc_kernel<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, fengtc::kSmemBytes) != cudaSuccess ||
        cudaFuncSetAttribute(fengtc::fengine_tc_kernel<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, fengtc::kSmemBytes) != cudaSuccess ||
        cudaFuncSetAttribute(fengtc::fengine_tc_kernel<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, fengtc::kSmemBytes) != cudaSuccess) {
        cudaGetLastError();
        cudaFree(d_tw);
        return nullptr;
    }
    st.d_tw = d_tw;
    st.ok = st.tried = true;
    return &st;
}

bool valid_geometry(int N, int P, int dtype) {
    return N >= 1 && (P == 1 || P == 2) && (dtype == CORR_CI8 || dtype == CORR_CF16);
}

// Triangular tile schedule of ONE channel for the direct feed, in real components u = 2m + {re, im}.
// Row block r covers u in [128 r, 128 r + 128); only columns up to the last station of the row block
// are needed (s_j <= s_i), cut into column blocks of 256.
void build_schedule_direct(int N, int P, std::vector<xtc::TileDesc>& v) {
    v.clear();
    const int M2 = 2 * N * P;
    for (int row0 = 0; row0 < M2; row0 += xtc::kTileRows) {
        const int row_end = (row0 + xtc::kTileRows < M2) ? row0 + xtc::kTileRows : M2;   // exclusive
        const int i_max = ((row_end - 1) / 2) / P;                                      // last station in the block
        const int need = (i_max + 1) * P * 2;                                           // columns u < need
        for (int col0 = 0; col0 < need; col0 += xtc::kTileCols) {
            int ncols = need - col0;
            if (ncols > xtc::kTileCols) ncols = xtc::kTileCols;
            ncols = (ncols + 15) & ~15;
            v.push_back(xtc::TileDesc{row0, col0, ncols, 0});
        }
    }
}

// Pair tiles of ONE channel: 256 x 256 blocks of G touching the lower station triangle, column-block major
// (tiles of one column block are adjacent, so clusters working at the same time share operands in L2).
void build_pair_tiles(int N, int P, std::vector<xtc::PairTile>& v) {
    v.clear();
    const int M2 = 2 * N * P;
    const int R = (M2 + xtc::kPairRows - 1) / xtc::kPairRows;
    for (int cb = 0; cb < R; ++cb)
        for (int rb = cb; rb < R; ++rb) v.push_back(xtc::PairTile{rb * xtc::kPairRows, cb * xtc::kPairRows});
}

// Rectangular cross-only plan: every 256 x 256 block of the [2 M_a] x [2 M_b] rectangle, column-block major.
void build_pair_tiles_rect(int Na, int Nb, int P, std::vector<xtc::PairTile>& v) {
    v.clear();
    const int Ra = (2 * Na * P + xtc::kPairRows - 1) / xtc::kPairRows;
    const int Rb = (2 * Nb * P + xtc::kPairRows - 1) / xtc::kPairRows;
    for (int cb = 0; cb < Rb; ++cb)
        for (int rb = 0; rb < Ra; ++rb) v.push_back(xtc::PairTile{rb * xtc::kPairRows, cb * xtc::kPairRows});
}

int resolve_kernel(const corr_plan* h) {
    if (!h->tma_ok) return CORR_KERNEL_SIMT;
    if (h->kernel != CORR_KERNEL_AUTO) return h->kernel;
    if (h->Nb) return h->max_clusters > 0 ? CORR_KERNEL_PAIR : CORR_KERNEL_SIMT;
    // PAIR vs SINGLE by executed MACs per sample and channel: a pair MAC costs ~0.72 of a 1-CTA MAC (half the operand
    // bytes from L2), but 256 x 256 tiles pad ragged 2M far more than 128-row tiles do.  Measured crossover (T = 2048,
    // N = 72 .. 384): PAIR wins iff pair MACs / single MACs < 1.39.
    if (h->max_clusters <= 0 || 2 * h->M < 256) return CORR_KERNEL_SINGLE;
    double single_macs = 0.0;
    for (const xtc::TileDesc& t : h->h_tiles) single_macs += static_cast<double>(xtc::kTileRows) * t.ncols;
    const double pair_macs = static_cast<double>(h->h_pair_tiles.size()) * xtc::kPairRows * xtc::kTileCols;
    return pair_macs < 1.39 * single_macs ? CORR_KERNEL_PAIR : CORR_KERNEL_SINGLE;
}

// sizes of the caller's buffers: always the WHOLE band (C_total channels), also for a window plan
size_t input_bytes(const corr_plan* h) {
    return static_cast<size_t>(h->T) * h->C_total * h->M * h->sample_bytes;
}
size_t output_bytes(const corr_plan* h) {
    return static_cast<size_t>(h->C_total) * h->B * h->P * h->P * 8;
}
size_t workspace_bytes(const corr_plan* h) {
    return 2 * static_cast<size_t>(h->C) * h->M * h->Tp * h->sample_bytes;
}
View device_view(const corr_plan* h) { return View{h->T, h->C, h->C_total, h->chan0, h->C_total, h->chan0}; }

// Tensor map of `ptr` viewed as [n_dump][n_time][c_total * 2 streams] real components, box [128 B][box_rows samples][1]:
// a box never crosses from one integration into the next, rows past an integration's end are zero-filled.  Encoded maps
// are cached per (pointer, shape): a caller cycling a few input buffers (config 4: four) pays the encode once each.
int get_map(corr_plan* h, const void* ptr, int streams, int c_total, int n_time, int n_dump, int box_rows,
            const CUtensorMap** out) {
    const MapKey key{ptr, streams, c_total, n_time, n_dump, box_rows};
    int victim = 0;
    for (int k = 0; k < kMapCache; ++k) {
        if (h->map_used[k] && h->map_key[k] == key) {
            h->map_used[k] = ++h->map_clock;
            *out = &h->map_val[k];
            return CORR_OK;
        }
        if (h->map_used[k] < h->map_used[victim]) victim = k;
    }
    const int elt = h->sample_bytes / 2;                       // bytes per real component
    const cuuint64_t W = static_cast<cuuint64_t>(c_total) * 2 * streams;
    cuuint64_t dims[3] = {W, static_cast<cuuint64_t>(n_time), static_cast<cuuint64_t>(n_dump)};
    cuuint64_t strides[2] = {W * elt, static_cast<cuuint64_t>(n_time) * W * elt};
    cuuint32_t box[3] = {static_cast<cuuint32_t>(128 / elt), static_cast<cuuint32_t>(box_rows), 1};
    cuuint32_t estr[3] = {1, 1, 1};
    const CUresult r = h->encode(&h->map_val[victim], elt == 1 ? CU_TENSOR_MAP_DATA_TYPE_UINT8 : CU_TENSOR_MAP_DATA_TYPE_FLOAT16,
                                 3, const_cast<void*>(ptr), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                 CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                                 CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        h->map_used[victim] = 0;
        return fail(h, CORR_ECUDA, "cuTensorMapEncodeTiled failed with CUresult %d", static_cast<int>(r));
    }
    h->map_key[victim] = key;
    h->map_used[victim] = ++h->map_clock;
    *out = &h->map_val[victim];
    return CORR_OK;
}

void fill_params(const corr_plan* h, const View& v, void* out, int accumulate, int n_dump, xtc::Params& prm) {
    prm.tiles = nullptr;
    prm.tiles_per_chan = 0;
    prm.n_tiles = 0;
    prm.n_station = h->N;
    prm.n_pol = h->P;
    prm.n_chan = v.n_chan;
    prm.n_time = v.n_time;
    prm.n_dump = n_dump;
    prm.M = h->M;
    prm.n_baseline = h->B;
    prm.n_station_b = h->Nb;
    prm.M_b = h->Mb;
    prm.out = out;
    prm.out_bytes = static_cast<unsigned long long>(n_dump) * v.c_total_out * h->B * h->P * h->P * 8;
    prm.accumulate = accumulate ? 1 : 0;
    // samples per TMEM accumulation pass: everything for int32 (exact); 1024 for fp32 (see xengine_tc.cuh)
    prm.k_chunk = h->dtype == CORR_CI8 ? (1 << 30) : xtc::kFloatChunk;
    prm.chan0 = v.chan0_in;
    prm.chan0_out = v.chan0_out;
    prm.n_chan_total = v.c_total_out;
    prm.n_stages = prm.stage_bytes = prm.b_chunks = 0;
}

int launch_direct(corr_plan* h, const View& v, const void* in, void* out, int accumulate, cudaStream_t st) {
    const CUtensorMap* map = nullptr;
    const int rc = get_map(h, in, h->M, v.c_total_in, v.n_time, 1,
                           h->dtype == CORR_CI8 ? xtc::Cfg<1>::kKStage : xtc::Cfg<2>::kKStage, &map);
    if (rc != CORR_OK) return rc;
    xtc::Params prm;
    fill_params(h, v, out, accumulate, 1, prm);
    prm.tiles = h->d_tiles;
    prm.tiles_per_chan = static_cast<int>(h->h_tiles.size());
    prm.n_tiles = static_cast<long long>(h->h_tiles.size()) * v.n_chan;
    {   // operand ring geometry: widest B of any tile, plus separate A chunks only if some tile is off the diagonal
        const int chunk_elems = h->dtype == CORR_CI8 ? 128 : 64;
        const int chunk_bytes = 128 * (h->dtype == CORR_CI8 ? xtc::Cfg<1>::kKStage : xtc::Cfg<2>::kKStage);
        int nb_max = 1;
        bool need_a = false;
        for (const xtc::TileDesc& t : h->h_tiles) {
            const int nb = (t.ncols + chunk_elems - 1) / chunk_elems;
            if (nb > nb_max) nb_max = nb;
            if (!(t.row0 >= t.col0 && t.row0 + xtc::kTileRows <= t.col0 + nb * chunk_elems)) need_a = true;
        }
        prm.b_chunks = nb_max;
        prm.stage_bytes = (nb_max + (need_a ? xtc::kTileRows / chunk_elems : 0)) * chunk_bytes;
        prm.n_stages = xtc::kRingBytes / prm.stage_bytes;
        if (prm.n_stages > xtc::kMaxStages) prm.n_stages = xtc::kMaxStages;
    }
    const long long grid = prm.n_tiles < h->sm_count ? prm.n_tiles : h->sm_count;
    if (h->dtype == CORR_CI8)
        xtc::xengine_direct_kernel<1><<<static_cast<unsigned>(grid), xtc::kNumThreads, xtc::kSmemBytes, st>>>(*map, prm);
    else
        xtc::xengine_direct_kernel<2><<<static_cast<unsigned>(grid), xtc::kNumThreads, xtc::kSmemBytes, st>>>(*map, prm);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail_cuda(h, e, "xengine_direct_kernel launch");
    h->last_launches += 1;
    return CORR_OK;
}

template <int kElt>
cudaError_t launch_pair_kernel(const CUtensorMap& tmap, const CUtensorMap& tmap_b, const xtc::PairParams& pp, unsigned clusters,
                               cudaStream_t st) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(clusters * 2);
    cfg.blockDim = dim3(xtc::kNumThreads);
    cfg.dynamicSmemBytes = xtc::kPairSmemBytes;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = 2;
    at[0].val.clusterDim.y = 1;
    at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, xtc::xengine_pair_kernel<kElt>, tmap, tmap_b, pp);
}

int launch_pair(corr_plan* h, const View& v, const void* in, const void* in_b, void* out, int accumulate, cudaStream_t st,
                int n_dump = 1) {
    const int box_rows = (h->dtype == CORR_CI8 ? xtc::kPairStageK<1> : xtc::kPairStageK<2>) / xtc::kPairBoxes;
    const CUtensorMap* map_a = nullptr;
    const CUtensorMap* map_b = nullptr;
    int rc = get_map(h, in, h->M, v.c_total_in, v.n_time, n_dump, box_rows, &map_a);
    if (rc == CORR_OK && h->Nb) rc = get_map(h, in_b, h->Mb, v.c_total_in, v.n_time, 1, box_rows, &map_b);
    if (rc != CORR_OK) return rc;
    if (!h->Nb) map_b = map_a;
    xtc::PairParams pp;
    fill_params(h, v, out, accumulate, n_dump, pp.base);
    pp.tiles = h->d_pair_tiles;
    pp.tiles_per_chan = static_cast<int>(h->h_pair_tiles.size());
    pp.n_tiles = static_cast<long long>(pp.tiles_per_chan) * v.n_chan * n_dump;
    if (pp.n_tiles > (1ll << 31) - 4096)
        return fail(h, CORR_EINVAL, "xengine_pair_kernel: %lld tiles exceed the tile feed's range", pp.n_tiles);
    const unsigned clusters = static_cast<unsigned>(pp.n_tiles < h->max_clusters ? pp.n_tiles : h->max_clusters);
    pp.sched_counter = h->d_sched + (h->sched_seq++ % kSchedRing);
    cudaError_t e = cudaMemsetAsync(pp.sched_counter, 0, sizeof(unsigned int), st);
    if (e != cudaSuccess) return fail_cuda(h, e, "tile-feed counter reset");
    e = h->dtype == CORR_CI8 ? launch_pair_kernel<1>(*map_a, *map_b, pp, clusters, st)
                             : launch_pair_kernel<2>(*map_a, *map_b, pp, clusters, st);
    if (e != cudaSuccess) return fail_cuda(h, e, "xengine_pair_kernel launch");
    h->last_launches += 1;
    return CORR_OK;
}

int launch_simt(corr_plan* h, const View& v, const void* in, const void* in_b, void* out, int accumulate, cudaStream_t st) {
    xsimt::Params prm;
    prm.in = in;
    prm.in_b = in_b;
    prm.n_station_b = h->Nb;
    prm.out = out;
    prm.n_station = h->N;
    prm.n_pol = h->P;
    prm.n_chan = v.n_chan;
    prm.n_time = v.n_time;
    prm.n_baseline = h->B;
    prm.n_vis = static_cast<long long>(v.n_chan) * h->B * h->P * h->P;
    prm.accumulate = accumulate ? 1 : 0;
    prm.chan0 = v.chan0_in;
    prm.n_chan_total = v.c_total_in;
    prm.chan0_out = v.chan0_out;
    long long blocks = (prm.n_vis + 127) / 128;
    const long long cap = static_cast<long long>(h->sm_count) * 16;
    if (blocks > cap) blocks = cap;
    if (h->dtype == CORR_CI8)
        xsimt::xengine_simt_kernel<false><<<static_cast<unsigned>(blocks), 128, 0, st>>>(prm);
    else
        xsimt::xengine_simt_kernel<true><<<static_cast<unsigned>(blocks), 128, 0, st>>>(prm);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail_cuda(h, e, "xengine_simt_kernel launch");
    h->last_launches += 1;
    return CORR_OK;
}

int launch_corner_turn(corr_plan* h, const void* in, void* ws, int n_planes, cudaStream_t st) {
    cturn::Params prm;
    prm.in = in;
    prm.ws = ws;
    prm.ws_rot = n_planes == 2 ? static_cast<uint8_t*>(ws) + workspace_bytes(h) / 2 : nullptr;
    prm.n_cm = static_cast<long long>(h->C) * h->M;
    prm.n_time = h->T;
    prm.n_time_pad = h->Tp;
    const unsigned gx = static_cast<unsigned>((prm.n_cm + cturn::kTileCm - 1) / cturn::kTileCm);
    if (h->dtype == CORR_CI8) {
        dim3 grid(gx, static_cast<unsigned>(h->Tp / 64));
        cturn::corner_turn_kernel<2><<<grid, cturn::kThreads, 0, st>>>(prm);
    } else {
        dim3 grid(gx, static_cast<unsigned>(h->Tp / 32));
        cturn::corner_turn_kernel<4><<<grid, cturn::kThreads, 0, st>>>(prm);
    }
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail_cuda(h, e, "corner_turn_kernel launch");
    h->last_launches += 1;
    return CORR_OK;
}

// One X-engine launch on a view, on whichever kernel the plan resolves to.
int launch_xengine(corr_plan* h, const View& v, const void* in, const void* in_b, void* out, int accumulate, cudaStream_t st) {
    switch (resolve_kernel(h)) {
        case CORR_KERNEL_PAIR: return launch_pair(h, v, in, in_b, out, accumulate, st);
        case CORR_KERNEL_SINGLE: return launch_direct(h, v, in, out, accumulate, st);
        default: return launch_simt(h, v, in, in_b, out, accumulate, st);
    }
}

}  // namespace

extern "C" {

long long corr_baseline_index(int i, int j) {
    if (j < 0 || j > i) return -1;
    return static_cast<long long>(i) * (i + 1) / 2 + j;
}

int corr_tile_schedule(int n_station, int n_pol, int dtype, int kernel, int* tiles3, int max_tiles) {
    if (!valid_geometry(n_station, n_pol, dtype) || max_tiles < 0 || (max_tiles > 0 && !tiles3)) return CORR_EINVAL;
    std::vector<int> flat;
    if (kernel == CORR_KERNEL_SINGLE) {
        std::vector<xtc::TileDesc> v;
        build_schedule_direct(n_station, n_pol, v);
        for (const xtc::TileDesc& t : v) { flat.push_back(t.row0); flat.push_back(t.col0); flat.push_back(t.ncols); }
    } else if (kernel == CORR_KERNEL_PAIR) {
        std::vector<xtc::PairTile> v;
        build_pair_tiles(n_station, n_pol, v);
        for (const xtc::PairTile& t : v) { flat.push_back(t.row0); flat.push_back(t.col0); flat.push_back(xtc::kTileCols); }
    } else {
        return CORR_EINVAL;
    }
    const int n = static_cast<int>(flat.size() / 3);
    for (int k = 0; k < n && k < max_tiles; ++k)
        for (int q = 0; q < 3; ++q) tiles3[3 * k + q] = flat[3 * k + q];
    return n;
}

static corr_handle create_plan(int n_station, int n_station_b, int n_pol, int n_chan_total, int chan0, int n_chan, int n_time,
                               int dtype) {
    g_create_error[0] = 0;
    if (!valid_geometry(n_station, n_pol, dtype) || n_station_b < 0 || n_chan < 1 || n_time < 1 || chan0 < 0 ||
        n_chan_total < 1 || static_cast<long long>(chan0) + n_chan > n_chan_total) {
        fail(nullptr, CORR_EINVAL, "corr_create: invalid geometry N=%d Nb=%d P=%d C=%d (window %d..+%d) T=%d dtype=%d", n_station,
             n_station_b, n_pol, n_chan_total, chan0, n_chan, n_time, dtype);
        return nullptr;
    }
    const long long M = static_cast<long long>(n_station) * n_pol;
    const long long Mb = static_cast<long long>(n_station_b) * n_pol;
    const long long W = static_cast<long long>(n_chan_total) * 2 * (M > Mb ? M : Mb);
    if (M > (1 << 20) || Mb > (1 << 20) || W > (1ll << 31) - 1024 || n_time > (1 << 24)) {
        fail(nullptr, CORR_EINVAL, "corr_create: geometry too large (N*P=%lld, C*2*N*P=%lld, T=%d)", M, W, n_time);
        return nullptr;
    }
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) {
        fail(nullptr, CORR_EUNSUPPORTED, "corr_create: no usable CUDA device (%s)", cudaGetErrorString(e));
        return nullptr;
    }
    cudaDeviceProp prop;
    e = cudaGetDeviceProperties(&prop, dev);
    if (e != cudaSuccess) {
        fail(nullptr, CORR_EUNSUPPORTED, "corr_create: cudaGetDeviceProperties: %s", cudaGetErrorString(e));
        return nullptr;
    }
    if (prop.major != 10 || prop.minor != 0) {       // the library carries sm_100a SASS only (no PTX): B200 / GB200
        fail(nullptr, CORR_EUNSUPPORTED, "corr_create: device %d (%s) is sm_%d%d; this library is built for sm_100a only",
             dev, prop.name, prop.major, prop.minor);
        return nullptr;
    }
    corr_plan* h = new (std::nothrow) corr_plan();
    if (!h) {
        fail(nullptr, CORR_ENOMEM, "corr_create: out of host memory");
        return nullptr;
    }
    h->N = n_station;
    h->P = n_pol;
    h->C = n_chan;
    h->C_total = n_chan_total;
    h->chan0 = chan0;
    h->T = n_time;
    h->dtype = dtype;
    h->M = static_cast<int>(M);
    h->Nb = n_station_b;
    h->Mb = static_cast<int>(Mb);
    h->B = n_station_b ? static_cast<long long>(n_station) * n_station_b       // rectangle: every (i, j)
                       : static_cast<long long>(n_station) * (n_station + 1) / 2;
    h->sample_bytes = dtype == CORR_CI8 ? 2 : 4;
    h->device = dev;
    h->sm_count = prop.multiProcessorCount;
    h->tma_ok = (M * h->sample_bytes) % 16 == 0 && (Mb * h->sample_bytes) % 16 == 0;
    h->t_total = 0;
    h->last_launches = 0;
    h->d_tiles = nullptr;
    h->d_pair_tiles = nullptr;
    h->kernel = CORR_KERNEL_AUTO;
    h->d_sched = nullptr;
    h->sched_seq = 0;
    h->max_clusters = 0;
    h->encode = nullptr;
    for (int k = 0; k < kMapCache; ++k) h->map_used[k] = 0;
    h->map_clock = 0;
    h->Tp = (n_time + 63) / 64 * 64;
    h->d_in_stage[0] = h->d_in_stage[1] = nullptr;
    h->d_out_stage = nullptr;
    h->host_sum_valid = false;
    h->st_h2d = h->st_run = h->st_d2h = nullptr;
    h->ev_h2d[0] = h->ev_h2d[1] = h->ev_run[0] = h->ev_run[1] = nullptr;
    h->err[0] = 0;

    build_schedule_direct(h->N, h->P, h->h_tiles);
    e = cudaMalloc(&h->d_tiles, h->h_tiles.size() * sizeof(xtc::TileDesc));
    if (e == cudaSuccess)
        e = cudaMemcpy(h->d_tiles, h->h_tiles.data(), h->h_tiles.size() * sizeof(xtc::TileDesc), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) {
        fail(nullptr, e == cudaErrorMemoryAllocation ? CORR_ENOMEM : CORR_ECUDA, "corr_create: tile table: %s",
             cudaGetErrorString(e));
        corr_destroy(h);
        return nullptr;
    }
    if (h->tma_ok) {
        h->encode = get_encode_fn();
        if (!h->encode) {
            fail(nullptr, CORR_ECUDA, "corr_create: cuTensorMapEncodeTiled entry point unavailable");
            corr_destroy(h);
            return nullptr;
        }
        e = cudaFuncSetAttribute(xtc::xengine_direct_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, xtc::kSmemBytes);
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(xtc::xengine_direct_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, xtc::kSmemBytes);
        if (e != cudaSuccess) {
            fail(nullptr, CORR_ECUDA, "corr_create: cudaFuncSetAttribute(smem): %s", cudaGetErrorString(e));
            corr_destroy(h);
            return nullptr;
        }
        e = cudaMalloc(&h->d_sched, kSchedRing * sizeof(unsigned int));
        if (e != cudaSuccess) {
            fail(nullptr, CORR_ENOMEM, "corr_create: tile-feed counters: %s", cudaGetErrorString(e));
            corr_destroy(h);
            return nullptr;
        }
        // CTA-pair kernel: tile table and the number of co-resident pairs (the persistent grid)
        if (h->Nb) build_pair_tiles_rect(h->N, h->Nb, h->P, h->h_pair_tiles);
        else build_pair_tiles(h->N, h->P, h->h_pair_tiles);
        const size_t bytes = h->h_pair_tiles.size() * sizeof(xtc::PairTile);
        e = cudaMalloc(&h->d_pair_tiles, bytes);
        if (e == cudaSuccess) e = cudaMemcpy(h->d_pair_tiles, h->h_pair_tiles.data(), bytes, cudaMemcpyHostToDevice);
        const void* fn_ptr = h->dtype == CORR_CI8 ? (const void*)xtc::xengine_pair_kernel<1> : (const void*)xtc::xengine_pair_kernel<2>;
        if (e == cudaSuccess) e = cudaFuncSetAttribute(fn_ptr, cudaFuncAttributeMaxDynamicSharedMemorySize, xtc::kPairSmemBytes);
        if (e == cudaSuccess) {
            cudaLaunchConfig_t cfg = {};
            cfg.gridDim = dim3(static_cast<unsigned>(h->sm_count / 2 * 2));
            cfg.blockDim = dim3(xtc::kNumThreads);
            cfg.dynamicSmemBytes = xtc::kPairSmemBytes;
            cudaLaunchAttribute at[1];
            at[0].id = cudaLaunchAttributeClusterDimension;
            at[0].val.clusterDim.x = 2;
            at[0].val.clusterDim.y = 1;
            at[0].val.clusterDim.z = 1;
            cfg.attrs = at;
            cfg.numAttrs = 1;
            int n = 0;
            if (cudaOccupancyMaxActiveClusters(&n, fn_ptr, &cfg) == cudaSuccess) h->max_clusters = n;
            else cudaGetLastError();          // pair kernel unavailable: resolve_kernel falls back
        }
        if (e != cudaSuccess) {
            fail(nullptr, e == cudaErrorMemoryAllocation ? CORR_ENOMEM : CORR_ECUDA, "corr_create: pair kernel setup: %s",
                 cudaGetErrorString(e));
            corr_destroy(h);
            return nullptr;
        }
    }
    return h;
}

corr_handle corr_create(int n_station, int n_pol, int n_chan, int n_time, int dtype) {
    return create_plan(n_station, 0, n_pol, n_chan, 0, n_chan, n_time, dtype);
}

corr_handle corr_create_window(int n_station, int n_pol, int n_chan_total, int chan0, int n_chan, int n_time, int dtype) {
    return create_plan(n_station, 0, n_pol, n_chan_total, chan0, n_chan, n_time, dtype);
}

corr_handle corr_create_cross(int n_station_a, int n_station_b, int n_pol, int n_chan, int n_time, int dtype) {
    if (n_station_b < 1) {
        g_create_error[0] = 0;
        fail(nullptr, CORR_EINVAL, "corr_create_cross: invalid geometry Na=%d Nb=%d", n_station_a, n_station_b);
        return nullptr;
    }
    return create_plan(n_station_a, n_station_b, n_pol, n_chan, 0, n_chan, n_time, dtype);
}

void corr_destroy(corr_handle h) {
    if (!h) return;
    if (h->d_tiles) cudaFree(h->d_tiles);
    if (h->d_sched) cudaFree(h->d_sched);
    if (h->d_pair_tiles) cudaFree(h->d_pair_tiles);
    for (int k = 0; k < 2; ++k) {
        if (h->d_in_stage[k]) cudaFree(h->d_in_stage[k]);
        if (h->ev_h2d[k]) cudaEventDestroy(h->ev_h2d[k]);
        if (h->ev_run[k]) cudaEventDestroy(h->ev_run[k]);
    }
    if (h->d_out_stage) cudaFree(h->d_out_stage);
    if (h->st_h2d) cudaStreamDestroy(h->st_h2d);
    if (h->st_run) cudaStreamDestroy(h->st_run);
    if (h->st_d2h) cudaStreamDestroy(h->st_d2h);
    delete h;
}

size_t corr_input_bytes(corr_handle h) { return h ? input_bytes(h) : 0; }
size_t corr_input_bytes_b(corr_handle h) { return h ? static_cast<size_t>(h->T) * h->C * h->Mb * h->sample_bytes : 0; }
size_t corr_output_bytes(corr_handle h) { return h ? output_bytes(h) : 0; }
size_t corr_workspace_bytes(corr_handle h) { return h ? workspace_bytes(h) : 0; }
int corr_workspace_time(corr_handle h) { return h ? h->Tp : 0; }
const char* corr_last_error(corr_handle h) { return h ? h->err : g_create_error; }
int corr_uses_tensor_cores(corr_handle h) { return h ? (resolve_kernel(h) != CORR_KERNEL_SIMT ? 1 : 0) : CORR_EINVAL; }
int corr_get_kernel(corr_handle h) { return h ? resolve_kernel(h) : CORR_EINVAL; }

int corr_set_kernel(corr_handle h, int kernel) {
    if (!h) return CORR_EINVAL;
    if (kernel < CORR_KERNEL_AUTO || kernel > CORR_KERNEL_SIMT) return fail(h, CORR_EINVAL, "corr_set_kernel: unknown kernel %d", kernel);
    if (kernel != CORR_KERNEL_AUTO && kernel != CORR_KERNEL_SIMT && !h->tma_ok)
        return fail(h, CORR_EUNSUPPORTED, "corr_set_kernel: per-channel row of %lld B is not a multiple of 16, only the SIMT kernel applies",
                    static_cast<long long>(h->M) * h->sample_bytes);
    if (h->Nb && kernel == CORR_KERNEL_SINGLE)
        return fail(h, CORR_EUNSUPPORTED, "corr_set_kernel: cross plans run on the PAIR or the SIMT kernel");
    if (kernel == CORR_KERNEL_PAIR && h->max_clusters <= 0)
        return fail(h, CORR_EUNSUPPORTED, "corr_set_kernel: no co-resident CTA pairs for the PAIR kernel on this device");
    h->kernel = kernel;
    return CORR_OK;
}
int corr_last_launch_count(corr_handle h) { return h ? h->last_launches : CORR_EINVAL; }

// tensor-core path (fp16 output and requantised int8 output): half tiles of 64 streams, the last one possibly ragged.  Taken
// when the output rows are 16-byte aligned (n_stream a multiple of 8: rows of n_stream x 2 or 4 bytes) and the padding of the
// ragged tile at most doubles the tensor work (n_stream >= 32 or a multiple of 64 ... 72 and 96 streams used to drop to the
// CUDA-core kernel at 0.40 of the HBM roof); below that the CUDA-core kernel wastes less.
static bool fengine_tc_applies(const void* out, int n_stream) {
    const int padded = (n_stream + fengtc::kTileStreams - 1) / fengtc::kTileStreams * fengtc::kTileStreams;
    return n_stream % 8 == 0 && padded <= 2 * n_stream && (reinterpret_cast<uintptr_t>(out) & 15) == 0;
}

static int run_fengine_tc(FengTcState* st, const void* in, void* out, int n_stream, long long n_spectra, bool int8_out, float scale,
                          cudaStream_t stream) {
    CUtensorMap map_raw;       // in viewed as [n_stream][n_spectra][256] bytes, box = 64 streams x 1 spectrum x 128 samples
    cuuint64_t dims[3] = {fengtc::kFft, static_cast<cuuint64_t>(n_spectra), static_cast<cuuint64_t>(n_stream)};
    cuuint64_t strides[2] = {fengtc::kFft, static_cast<cuuint64_t>(n_spectra) * fengtc::kFft};
    cuuint32_t box[3] = {fengtc::kFft / 2, 1, fengtc::kTileStreams};
    cuuint32_t estr[3] = {1, 1, 1};
    const CUresult r = st->encode(&map_raw, CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, const_cast<void*>(in), dims, strides, box, estr,
                                  CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(nullptr, CORR_ECUDA, "corr_fengine: cuTensorMapEncodeTiled failed with CUresult %d", static_cast<int>(r));
    fengtc::Params prm;
    prm.out = out;
    prm.scale = scale;
    prm.tw = static_cast<const uint4*>(st->d_tw);
    prm.n_stream = n_stream;
    prm.n_spectra = n_spectra;
    prm.n_half = n_spectra * ((n_stream + fengtc::kTileStreams - 1) / fengtc::kTileStreams);
    prm.n_tiles = (prm.n_half + 1) / 2;
    const long long grid = prm.n_tiles < st->sm_count ? prm.n_tiles : st->sm_count;
    const unsigned g = static_cast<unsigned>(grid);
    const bool ragged = n_stream % fengtc::kTileStreams != 0;
    if (int8_out && ragged) fengtc::fengine_tc_kernel<true, true><<<g, fengtc::kThreads, fengtc::kSmemBytes, stream>>>(map_raw, prm);
    else if (int8_out) fengtc::fengine_tc_kernel<true, false><<<g, fengtc::kThreads, fengtc::kSmemBytes, stream>>>(map_raw, prm);
    else if (ragged) fengtc::fengine_tc_kernel<false, true><<<g, fengtc::kThreads, fengtc::kSmemBytes, stream>>>(map_raw, prm);
    else fengtc::fengine_tc_kernel<false, false><<<g, fengtc::kThreads, fengtc::kSmemBytes, stream>>>(map_raw, prm);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail_cuda(nullptr, e, "fengine_tc_kernel launch");
    return CORR_OK;
}

static int run_fengine(const void* in, void* out, int n_stream, long long n_spectra, bool int8_out, float scale, void* stream,
                       bool allow_tc = true) {
    g_create_error[0] = 0;
    if (!in || !out || n_stream < 1 || n_spectra < 1 || n_spectra > 0x7fffffffLL || (int8_out && !(scale > 0.0f)))
        return fail(nullptr, CORR_EINVAL, "corr_fengine: invalid arguments (n_stream=%d, n_spectra=%lld)", n_stream, n_spectra);
    if ((reinterpret_cast<uintptr_t>(in) & 15) || (reinterpret_cast<uintptr_t>(out) & (int8_out ? 1 : 3)))
        return fail(nullptr, CORR_EINVAL, "corr_fengine: `in` must be 16-byte and `out` element aligned");
    if (allow_tc && fengine_tc_applies(out, n_stream)) {
        FengTcState* st = fengine_tc_state();
        if (st) return run_fengine_tc(st, in, out, n_stream, n_spectra, int8_out, scale, static_cast<cudaStream_t>(stream));
    }
    feng::Params prm;
    prm.in = static_cast<const int8_t*>(in);
    prm.out = out;
    prm.n_stream = n_stream;
    prm.n_spectra = n_spectra;
    prm.scale = scale;
    const long long n_sb = (n_stream + feng::kStreamsPerBlock - 1) / feng::kStreamsPerBlock;
    const long long n_ab = (n_spectra + feng::kSpectraPerBlock - 1) / feng::kSpectraPerBlock;
    if (n_sb * n_ab > 0x7fffffffLL) return fail(nullptr, CORR_EINVAL, "corr_fengine: problem too large for one launch");
    const dim3 grid(static_cast<unsigned>(n_sb * n_ab));
    if (int8_out) feng::fengine_kernel<true><<<grid, feng::kThreads, 0, static_cast<cudaStream_t>(stream)>>>(prm);
    else feng::fengine_kernel<false><<<grid, feng::kThreads, 0, static_cast<cudaStream_t>(stream)>>>(prm);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail_cuda(nullptr, e, "fengine_kernel launch");
    return CORR_OK;
}

int corr_fengine(const void* in, void* out, int n_stream, long long n_spectra, void* stream) {
    return run_fengine(in, out, n_stream, n_spectra, false, 1.0f, stream);
}

int corr_fengine_ci8(const void* in, void* out, int n_stream, long long n_spectra, float scale, void* stream) {
    return run_fengine(in, out, n_stream, n_spectra, true, scale, stream);
}

int corr_fengine_simt(const void* in, void* out, int n_stream, long long n_spectra, void* stream) {
    return run_fengine(in, out, n_stream, n_spectra, false, 1.0f, stream, false);
}

int corr_fengine_uses_tensor_cores(int n_stream, const void* out) {
    // the same two conditions run_fengine applies, in the same order: geometry / alignment, then the device's state
    return fengine_tc_applies(out, n_stream) && fengine_tc_state() != nullptr ? 1 : 0;
}

int corr_corner_turn(corr_handle h, const void* in, void* ws, void* stream) {
    return corr_corner_turn_planes(h, in, ws, 2, stream);
}

int corr_corner_turn_planes(corr_handle h, const void* in, void* ws, int n_planes, void* stream) {
    if (!h) return CORR_EINVAL;
    if (n_planes != 1 && n_planes != 2) return fail(h, CORR_EINVAL, "corr_corner_turn_planes: n_planes must be 1 or 2");
    if (h->Nb || h->C != h->C_total) return fail(h, CORR_EINVAL, "corr_corner_turn: not available on cross or window plans");
    if (!in || !ws) return fail(h, CORR_EINVAL, "corr_corner_turn: NULL pointer");
    if ((reinterpret_cast<uintptr_t>(in) & 15) || (reinterpret_cast<uintptr_t>(ws) & 127))
        return fail(h, CORR_EINVAL, "corr_corner_turn: `in` must be 16-byte and `ws` 128-byte aligned");
    if (!h->tma_ok)
        return fail(h, CORR_EUNSUPPORTED, "corr_corner_turn: per-channel row of %lld B is not a multiple of 16",
                    static_cast<long long>(h->M) * h->sample_bytes);
    h->last_launches = 0;
    return launch_corner_turn(h, in, ws, n_planes, static_cast<cudaStream_t>(stream));
}

static int run_xengine(corr_handle h, const void* in, const void* in_b, void* out, int accumulate, void* stream) {
    if (!in || !out) return fail(h, CORR_EINVAL, "corr_xengine: NULL pointer");
    if ((reinterpret_cast<uintptr_t>(in) & 15) || (reinterpret_cast<uintptr_t>(out) & 15))
        return fail(h, CORR_EINVAL, "corr_xengine: `in` and `out` must be 16-byte aligned");
    const long long t_next = accumulate ? h->t_total + h->T : h->T;
    if (h->dtype == CORR_CI8 && t_next > kMaxIntegrationCi8)
        return fail(h, CORR_EOVERFLOW, "corr_xengine: integrating %lld samples would overflow int32 (limit %lld)", t_next,
                    kMaxIntegrationCi8);
    h->last_launches = 0;
    const int rc = launch_xengine(h, device_view(h), in, in_b, out, accumulate, static_cast<cudaStream_t>(stream));
    if (rc == CORR_OK) h->t_total = t_next;
    return rc;
}

int corr_xengine(corr_handle h, const void* in, void* out, int accumulate, void* stream) {
    if (!h) return CORR_EINVAL;
    if (h->Nb) return fail(h, CORR_EINVAL, "corr_xengine: this is a cross plan (corr_create_cross); call corr_xengine_cross");
    return run_xengine(h, in, nullptr, out, accumulate, stream);
}

int corr_xengine_dumps(corr_handle h, const void* in, void* out, int n_dump, void* stream) {
    if (!h) return CORR_EINVAL;
    if (h->Nb) return fail(h, CORR_EINVAL, "corr_xengine_dumps: not available on cross plans");
    if (!in || !out) return fail(h, CORR_EINVAL, "corr_xengine_dumps: NULL pointer");
    if ((reinterpret_cast<uintptr_t>(in) & 15) || (reinterpret_cast<uintptr_t>(out) & 15))
        return fail(h, CORR_EINVAL, "corr_xengine_dumps: `in` and `out` must be 16-byte aligned");
    if (n_dump < 1 || h->T % n_dump)
        return fail(h, CORR_EINVAL, "corr_xengine_dumps: n_dump = %d must divide n_time = %d", n_dump, h->T);
    const int Ts = h->T / n_dump;
    if (h->dtype == CORR_CI8 && Ts > kMaxIntegrationCi8)
        return fail(h, CORR_EOVERFLOW, "corr_xengine_dumps: integrating %d samples would overflow int32", Ts);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    h->last_launches = 0;       // (the running-integration count t_total of corr_xengine is not touched: dumps never accumulate)
    View v = device_view(h);
    v.n_time = Ts;
    if (resolve_kernel(h) != CORR_KERNEL_SIMT && h->max_clusters > 0)
        return launch_pair(h, v, in, nullptr, out, 0, st, n_dump);        // any TMA-addressable geometry runs on the pair kernel
    // SIMT: one launch per integration on slices of `in` and `out`
    int rc = CORR_OK;
    for (int d = 0; d < n_dump && rc == CORR_OK; ++d)
        rc = launch_simt(h, v, static_cast<const uint8_t*>(in) + d * (input_bytes(h) / n_dump), nullptr,
                         static_cast<uint8_t*>(out) + d * output_bytes(h), 0, st);
    return rc;
}

int corr_xengine_cross(corr_handle h, const void* in_a, const void* in_b, void* out, int accumulate, void* stream) {
    if (!h) return CORR_EINVAL;
    if (!h->Nb) return fail(h, CORR_EINVAL, "corr_xengine_cross: this is not a cross plan; call corr_xengine");
    if (!in_b || (reinterpret_cast<uintptr_t>(in_b) & 15))
        return fail(h, CORR_EINVAL, "corr_xengine_cross: `in_b` must be a non-NULL, 16-byte aligned device pointer");
    return run_xengine(h, in_a, in_b, out, accumulate, stream);
}

// Host-buffer entry point: the plan's channels are cut into up to kHostWindows windows that flow through a three-stage
// pipeline on three streams -- H2D of window w+1 (a strided 2-D copy straight out of the caller's [T][C][M] buffer into
// one of two compact staging slots), the X-engine on window w (reading the slot, writing its slab of the device-resident
// running sum), D2H of window w-1's slab -- so the PCIe link runs in both directions while the kernel computes.
int corr_xengine_host(corr_handle h, const void* in_host, void* out_host, int accumulate) {
    if (!h) return CORR_EINVAL;
    if (h->Nb) return fail(h, CORR_EINVAL, "corr_xengine_host: not available on cross plans");
    if (!in_host) return fail(h, CORR_EINVAL, "corr_xengine_host: NULL input pointer");
    const long long t_next = accumulate ? h->t_total + h->T : h->T;
    if (h->dtype == CORR_CI8 && t_next > kMaxIntegrationCi8)
        return fail(h, CORR_EOVERFLOW, "corr_xengine_host: integrating %lld samples would overflow int32 (limit %lld)", t_next,
                    kMaxIntegrationCi8);
    cudaError_t e = cudaSuccess;
    const int n_win = h->C < kHostWindows ? h->C : kHostWindows;
    const int win_max = (h->C + n_win - 1) / n_win;
    const size_t chan_in_bytes = static_cast<size_t>(h->M) * h->sample_bytes;             // one channel of one time sample
    const size_t chan_out_bytes = static_cast<size_t>(h->B) * h->P * h->P * 8;            // one channel's visibilities
    if (!h->st_h2d) {
        e = cudaStreamCreateWithFlags(&h->st_h2d, cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&h->st_run, cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&h->st_d2h, cudaStreamNonBlocking);
        for (int k = 0; k < 2 && e == cudaSuccess; ++k) {
            e = cudaEventCreateWithFlags(&h->ev_h2d[k], cudaEventDisableTiming);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&h->ev_run[k], cudaEventDisableTiming);
        }
        if (e != cudaSuccess) return fail_cuda(h, e, "corr_xengine_host: streams / events");
    }
    for (int k = 0; k < 2; ++k)
        if (!h->d_in_stage[k]) {
            e = cudaMalloc(&h->d_in_stage[k], static_cast<size_t>(h->T) * win_max * chan_in_bytes);
            if (e != cudaSuccess) return fail(h, CORR_ENOMEM, "corr_xengine_host: input staging: %s", cudaGetErrorString(e));
        }
    if (accumulate && !h->host_sum_valid)
        return fail(h, CORR_EINVAL, "corr_xengine_host: accumulate without a complete previous integration on this handle "
                                    "(no earlier call, or the last one failed part-way)");
    if (!h->d_out_stage) {
        e = cudaMalloc(&h->d_out_stage, static_cast<size_t>(h->C) * chan_out_bytes);
        if (e != cudaSuccess) return fail(h, CORR_ENOMEM, "corr_xengine_host: output staging: %s", cudaGetErrorString(e));
    }
    h->last_launches = 0;
    h->host_sum_valid = false;            // until every window of this call has gone through
    const uint8_t* src = static_cast<const uint8_t*>(in_host);
    uint8_t* dst = static_cast<uint8_t*>(out_host);
    const int base = h->C / n_win, extra = h->C % n_win;
    // A failure part-way leaves copies queued that still read `in_host` / write `out_host`, and some windows of the running
    // sum already updated: drain all three streams before returning (the caller may free its buffers right away) and leave
    // the running sum marked invalid, so that a retry cannot double-count the windows that did go through.
    auto bail = [&](int code) {
        cudaStreamSynchronize(h->st_h2d);
        cudaStreamSynchronize(h->st_run);
        cudaStreamSynchronize(h->st_d2h);
        cudaGetLastError();
        return code;
    };
    int c0 = 0;
    for (int w = 0; w < n_win; ++w) {
        const int wn = base + (w < extra ? 1 : 0);
        const int slot = w & 1;
        if (w >= 2) {                                     // the kernel of window w - 2 has finished reading this slot
            e = cudaStreamWaitEvent(h->st_h2d, h->ev_run[slot], 0);
            if (e != cudaSuccess) return bail(fail_cuda(h, e, "corr_xengine_host: wait for the staging slot"));
        }
        e = cudaMemcpy2DAsync(h->d_in_stage[slot], wn * chan_in_bytes, src + static_cast<size_t>(h->chan0 + c0) * chan_in_bytes,
                              static_cast<size_t>(h->C_total) * chan_in_bytes, wn * chan_in_bytes, h->T, cudaMemcpyHostToDevice,
                              h->st_h2d);
        if (e == cudaSuccess) e = cudaEventRecord(h->ev_h2d[slot], h->st_h2d);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(h->st_run, h->ev_h2d[slot], 0);
        if (e != cudaSuccess) return bail(fail_cuda(h, e, "corr_xengine_host: H2D copy"));
        const View v{h->T, wn, wn, 0, h->C, c0};
        const int rc = launch_xengine(h, v, h->d_in_stage[slot], nullptr, h->d_out_stage, accumulate, h->st_run);
        if (rc != CORR_OK) return bail(rc);
        e = cudaEventRecord(h->ev_run[slot], h->st_run);
        if (e == cudaSuccess && dst) {
            e = cudaStreamWaitEvent(h->st_d2h, h->ev_run[slot], 0);
            if (e == cudaSuccess)
                e = cudaMemcpyAsync(dst + static_cast<size_t>(h->chan0 + c0) * chan_out_bytes,
                                    static_cast<uint8_t*>(h->d_out_stage) + static_cast<size_t>(c0) * chan_out_bytes,
                                    wn * chan_out_bytes, cudaMemcpyDeviceToHost, h->st_d2h);
        }
        if (e != cudaSuccess) return bail(fail_cuda(h, e, "corr_xengine_host: D2H copy"));
        c0 += wn;
    }
    e = cudaStreamSynchronize(h->st_run);
    if (e == cudaSuccess) e = cudaStreamSynchronize(h->st_d2h);
    if (e == cudaSuccess) e = cudaStreamSynchronize(h->st_h2d);
    if (e != cudaSuccess) return bail(fail_cuda(h, e, "corr_xengine_host: stream synchronize"));
    h->host_sum_valid = true;
    h->t_total = t_next;
    return CORR_OK;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------------------------------
// corr_xengine_static: the CTA-pair X-engine for callers that must not allocate device memory (include/corr.h).
//
// The pair kernel needs two pieces of global memory besides the caller's input and output: the per-channel tile table
// it walks and the 4-byte tile-feed counter its clusters claim work from.  A handle gets both from cudaMalloc in
// corr_create.  Here they live in ONE file-scope device array that is part of the library image, so no call on this path
// ever asks the driver for memory: every GPU that loads libcorr.so carries these kStaticScratchBytes (16.5 KB) until the
// process exits, used or not.
//
// g_static_scratch is a DEVICE symbol.  In host code its name is only a host-side shadow of the symbol, not a device
// address: handing `g_static_scratch` itself to a kernel would make the kernel fault (or, on systems where the GPU can
// reach host memory, quietly work on the wrong memory).  The device address is looked up once per device with
// cudaGetSymbolAddress (static_state below) and only that pointer is passed to kernels.  Device code in this file
// (static_prepare_kernel) may name the array directly.
namespace {

constexpr int kStaticMaxBlocks = CORR_STATIC_MAX_STREAMS * 2 / xtc::kPairRows;            // 64 row blocks of 256 components
constexpr int kStaticMaxTiles = kStaticMaxBlocks * (kStaticMaxBlocks + 1) / 2;            // 2080 pair tiles per channel
constexpr int kStaticCounterWords = 64;      // word 0 is the tile-feed counter; the rest pads the table to a 256-byte boundary
constexpr int kStaticWords = kStaticCounterWords + 2 * kStaticMaxTiles;
constexpr size_t kStaticScratchBytes = sizeof(unsigned int) * kStaticWords;
static_assert(sizeof(xtc::PairTile) == 2 * sizeof(unsigned int), "tile table entry");

static __device__ __align__(256) unsigned int g_static_scratch[kStaticWords];

// Prepares the shared scratch for one launch, on the launch's own stream: the array still holds whatever the previous
// call left there (a counter that has run past its tile count, a table for another station count), so the counter is
// cleared and the table rewritten every time.  Same order as build_pair_tiles: column-block major, row block >= column block.
__global__ void static_prepare_kernel(int n_blocks) {
    if (blockIdx.x == 0 && threadIdx.x == 0) g_static_scratch[0] = 0u;
    xtc::PairTile* tiles = reinterpret_cast<xtc::PairTile*>(g_static_scratch + kStaticCounterWords);
    for (int k = blockIdx.x * blockDim.x + threadIdx.x; k < n_blocks * n_blocks; k += gridDim.x * blockDim.x) {
        const int cb = k / n_blocks, rb = k - cb * n_blocks;
        if (rb < cb) continue;
        const int idx = cb * n_blocks - cb * (cb - 1) / 2 + (rb - cb);
        tiles[idx] = xtc::PairTile{rb * xtc::kPairRows, cb * xtc::kPairRows};
    }
}

struct StaticState {
    bool ready = false;
    unsigned int* scratch = nullptr;        // DEVICE address of g_static_scratch on this device
    EncodeTiledFn encode = nullptr;
    int sm_count = 0;
    int max_clusters[2] = {0, 0};           // co-resident CTA pairs of the ci8 / cf16 pair kernel
};
std::mutex g_static_mutex;
StaticState g_static[64];

// One-time set-up for the CURRENT device (looked up again on every call, done once).  Nothing here allocates device
// memory: it resolves the scratch array's device address, raises the pair kernels' shared-memory limit and asks how many
// CTA pairs fit on the GPU.  `ready` is set only after everything succeeded, so a transient failure is retried by the next call.
int static_state(StaticState** out) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(nullptr, CORR_EUNSUPPORTED, "corr_xengine_static: no usable CUDA device (%s)", cudaGetErrorString(e));
    if (dev < 0 || dev >= 64) return fail(nullptr, CORR_EUNSUPPORTED, "corr_xengine_static: device ordinal %d out of range", dev);
    std::lock_guard<std::mutex> lock(g_static_mutex);
    StaticState& st = g_static[dev];
    if (!st.ready) {
        int major = 0, minor = 0, sms = 0;
        e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
        if (e == cudaSuccess) e = cudaDeviceGetAttribute(&minor, cudaDevAttrComputeCapabilityMinor, dev);
        if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) return fail(nullptr, CORR_EUNSUPPORTED, "corr_xengine_static: device query: %s", cudaGetErrorString(e));
        if (major != 10 || minor != 0)
            return fail(nullptr, CORR_EUNSUPPORTED, "corr_xengine_static: device %d is sm_%d%d; this library is built for sm_100a only",
                        dev, major, minor);
        unsigned int* ptr = nullptr;
        e = cudaGetSymbolAddress(reinterpret_cast<void**>(&ptr), g_static_scratch);
        if (e != cudaSuccess || !ptr) {
            cudaGetLastError();
            return fail(nullptr, CORR_ECUDA, "corr_xengine_static: cudaGetSymbolAddress(scratch): %s", cudaGetErrorString(e));
        }
        EncodeTiledFn enc = get_encode_fn();
        if (!enc) return fail(nullptr, CORR_ECUDA, "corr_xengine_static: cuTensorMapEncodeTiled entry point unavailable");
        int clusters[2] = {0, 0};
        for (int k = 0; k < 2; ++k) {
            const void* fn_ptr = k == 0 ? (const void*)xtc::xengine_pair_kernel<1> : (const void*)xtc::xengine_pair_kernel<2>;
            e = cudaFuncSetAttribute(fn_ptr, cudaFuncAttributeMaxDynamicSharedMemorySize, xtc::kPairSmemBytes);
            if (e != cudaSuccess) {
                cudaGetLastError();
                return fail(nullptr, CORR_ECUDA, "corr_xengine_static: cudaFuncSetAttribute(smem): %s", cudaGetErrorString(e));
            }
            cudaLaunchConfig_t cfg = {};
            cfg.gridDim = dim3(static_cast<unsigned>(sms / 2 * 2));
            cfg.blockDim = dim3(xtc::kNumThreads);
            cfg.dynamicSmemBytes = xtc::kPairSmemBytes;
            cudaLaunchAttribute at[1];
            at[0].id = cudaLaunchAttributeClusterDimension;
            at[0].val.clusterDim.x = 2;
            at[0].val.clusterDim.y = 1;
            at[0].val.clusterDim.z = 1;
            cfg.attrs = at;
            cfg.numAttrs = 1;
            e = cudaOccupancyMaxActiveClusters(&clusters[k], fn_ptr, &cfg);
            if (e != cudaSuccess || clusters[k] <= 0) {
                cudaGetLastError();
                return fail(nullptr, CORR_EUNSUPPORTED, "corr_xengine_static: no co-resident CTA pairs for the pair kernel on device %d", dev);
            }
        }
        st.scratch = ptr;
        st.encode = enc;
        st.sm_count = sms;
        st.max_clusters[0] = clusters[0];
        st.max_clusters[1] = clusters[1];
        st.ready = true;
    }
    *out = &st;
    return CORR_OK;
}

}  // namespace

extern "C" {

size_t corr_static_scratch_bytes(void) { return kStaticScratchBytes; }

int corr_xengine_static(int n_station, int n_pol, int n_chan, int n_time, int dtype, const void* in, void* out, int accumulate,
                        void* stream) {
    g_create_error[0] = 0;
    // ---- arguments first: nothing below this block is reached (and no CUDA call is made) for a rejected geometry ----
    if (!valid_geometry(n_station, n_pol, dtype) || n_chan < 1 || n_time < 1)
        return fail(nullptr, CORR_EINVAL, "corr_xengine_static: invalid geometry N=%d P=%d C=%d T=%d dtype=%d", n_station, n_pol,
                    n_chan, n_time, dtype);
    const long long M = static_cast<long long>(n_station) * n_pol;
    if (M > CORR_STATIC_MAX_STREAMS)
        return fail(nullptr, CORR_EINVAL,
                    "corr_xengine_static: n_station * n_pol = %lld exceeds CORR_STATIC_MAX_STREAMS = %d, the largest tile table "
                    "the library's built-in scratch array holds (%d tiles per channel); use corr_create / corr_xengine",
                    M, CORR_STATIC_MAX_STREAMS, kStaticMaxTiles);
    const int sample_bytes = dtype == CORR_CI8 ? 2 : 4;
    if (static_cast<long long>(n_chan) * 2 * M > (1ll << 31) - 1024 || n_time > (1 << 24))
        return fail(nullptr, CORR_EINVAL, "corr_xengine_static: geometry too large (C*2*N*P=%lld, T=%d)",
                    static_cast<long long>(n_chan) * 2 * M, n_time);
    if ((M * sample_bytes) % 16 != 0)
        return fail(nullptr, CORR_EUNSUPPORTED,
                    "corr_xengine_static: per-channel row of %lld B is not a multiple of 16 (TMA cannot address it); use corr_create",
                    M * sample_bytes);
    if (dtype == CORR_CI8 && n_time > kMaxIntegrationCi8)
        return fail(nullptr, CORR_EOVERFLOW, "corr_xengine_static: integrating %d samples would overflow int32 (limit %lld)", n_time,
                    kMaxIntegrationCi8);
    if (!in || !out) return fail(nullptr, CORR_EINVAL, "corr_xengine_static: NULL pointer");
    if ((reinterpret_cast<uintptr_t>(in) & 15) || (reinterpret_cast<uintptr_t>(out) & 15))
        return fail(nullptr, CORR_EINVAL, "corr_xengine_static: `in` and `out` must be 16-byte aligned");
    const int n_blocks = static_cast<int>((2 * M + xtc::kPairRows - 1) / xtc::kPairRows);
    const int tiles_per_chan = n_blocks * (n_blocks + 1) / 2;
    const long long n_tiles = static_cast<long long>(tiles_per_chan) * n_chan;
    if (n_blocks > kStaticMaxBlocks || tiles_per_chan > kStaticMaxTiles)        // (implied by the stream limit; kept as the array's own guard)
        return fail(nullptr, CORR_EINVAL, "corr_xengine_static: %d tiles per channel exceed the scratch array's %d", tiles_per_chan,
                    kStaticMaxTiles);
    if (n_tiles > (1ll << 31) - 4096)
        return fail(nullptr, CORR_EINVAL, "corr_xengine_static: %lld tiles exceed the tile feed's range", n_tiles);

    StaticState* st = nullptr;
    int rc = static_state(&st);
    if (rc != CORR_OK) return rc;

    // a plan on the stack, never a heap or device allocation: only the fields fill_params / get_map read
    corr_plan plan{};
    plan.N = n_station;
    plan.P = n_pol;
    plan.C = plan.C_total = n_chan;
    plan.T = n_time;
    plan.dtype = dtype;
    plan.M = static_cast<int>(M);
    plan.B = static_cast<long long>(n_station) * (n_station + 1) / 2;
    plan.sample_bytes = sample_bytes;
    plan.encode = st->encode;
    const View v{n_time, n_chan, n_chan, 0, n_chan, 0};
    const int box_rows = (dtype == CORR_CI8 ? xtc::kPairStageK<1> : xtc::kPairStageK<2>) / xtc::kPairBoxes;
    const CUtensorMap* map = nullptr;
    rc = get_map(&plan, in, plan.M, n_chan, n_time, 1, box_rows, &map);        // host-side encode into plan.map_val[]
    if (rc != CORR_OK) {
        fail(nullptr, rc, "corr_xengine_static: %s", plan.err);
        return rc;
    }
    xtc::PairParams pp;
    fill_params(&plan, v, out, accumulate, 1, pp.base);
    pp.sched_counter = st->scratch;                                                        // DEVICE addresses inside the
    pp.tiles = reinterpret_cast<const xtc::PairTile*>(st->scratch + kStaticCounterWords);  // static scratch array
    pp.tiles_per_chan = tiles_per_chan;
    pp.n_tiles = n_tiles;
    const int max_clusters = st->max_clusters[dtype == CORR_CI8 ? 0 : 1];
    const unsigned clusters = static_cast<unsigned>(n_tiles < max_clusters ? n_tiles : max_clusters);

    cudaStream_t cs = static_cast<cudaStream_t>(stream);
    const int cells = n_blocks * n_blocks;
    static_prepare_kernel<<<(cells + 255) / 256, 256, 0, cs>>>(n_blocks);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail_cuda(nullptr, e, "corr_xengine_static: scratch preparation launch");
    e = dtype == CORR_CI8 ? launch_pair_kernel<1>(*map, *map, pp, clusters, cs) : launch_pair_kernel<2>(*map, *map, pp, clusters, cs);
    if (e != cudaSuccess) return fail_cuda(nullptr, e, "corr_xengine_static: xengine_pair_kernel launch");
    return CORR_OK;
}

}  // extern "C"
