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
#include <cstring>
#include <new>
#include <vector>

#include "corner_turn.cuh"
#include "fengine.cuh"
#include "xengine_simt.cuh"
#include "xengine_tc.cuh"
#include "xengine_pair.cuh"

namespace {

constexpr long long kMaxIntegrationCi8 = 65535;
constexpr unsigned kSchedRing = 256;            // launches in flight on different streams never share a feed counter   // 2 * 128^2 * T_total <= 2^31 - 1

thread_local char g_create_error[512] = "";

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

}  // namespace

struct corr_plan {
    int N, P, C, T, dtype;
    int M;                 // N * P
    int Nb, Mb;            // rectangular cross-only plan (corr_create_cross): stations / streams of group B; 0 = HERK
    long long B;           // N (N + 1) / 2
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
    std::vector<xtc::PairGroup> h_groups[2];   // [0]: one pair per cluster, [1]: two pairs per cluster (multicast)
    xtc::PairGroup* d_groups[2];
    unsigned int* d_sched;                     // ring of tile-feed counters, one per launch (kSchedRing)
    unsigned int sched_seq;
    int max_clusters[2];                       // co-resident clusters of 2 / 4 CTAs (cudaOccupancyMaxActiveClusters)
    EncodeTiledFn encode;

    CUtensorMap tmap_in;     // 1-CTA kernel: box [128 B][Cfg::kKStage samples]
    CUtensorMap tmap_pair;   // pair kernels: box [128 B][kPairStageK / kPairBoxes samples]
    const void* tmap_in_ptr;
    int tmap_dumps;          // n_dump the pair tensor map was encoded for
    CUtensorMap tmap_b;      // cross plans: group B, pair-kernel box
    const void* tmap_b_ptr;

    // corner-turn feed
    int Tp;                // padded time extent of the workspace

    // corr_xengine_host staging
    void* d_in_stage;
    void* d_out_stage;
    cudaStream_t own_stream;

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

// Groups of ONE channel.  pairs_per_cluster == 1: one tile per group.  == 2: two tiles sharing their column
// block (B multicast); the odd tile out of each column block lies in the last row block, and those are joined
// two by two (A multicast); a last single tile is duplicated (computed twice, written once).
void build_groups(int N, int P, int pairs_per_cluster, std::vector<xtc::PairGroup>& g) {
    g.clear();
    const int M2 = 2 * N * P;
    const int R = (M2 + xtc::kPairRows - 1) / xtc::kPairRows;
    if (pairs_per_cluster == 1) {
        std::vector<xtc::PairTile> t;
        build_pair_tiles(N, P, t);
        for (const xtc::PairTile& x : t) g.push_back(xtc::PairGroup{{x, x}, 0, 0});
        return;
    }
    std::vector<xtc::PairTile> odd;
    for (int cb = 0; cb < R; ++cb) {
        int rb = cb;
        for (; rb + 1 < R; rb += 2)
            g.push_back(xtc::PairGroup{{{rb * xtc::kPairRows, cb * xtc::kPairRows}, {(rb + 1) * xtc::kPairRows, cb * xtc::kPairRows}}, 2, 0});
        if (rb < R) odd.push_back(xtc::PairTile{rb * xtc::kPairRows, cb * xtc::kPairRows});
    }
    size_t k = 0;
    for (; k + 1 < odd.size(); k += 2) g.push_back(xtc::PairGroup{{odd[k], odd[k + 1]}, 1, 0});
    if (k < odd.size()) g.push_back(xtc::PairGroup{{odd[k], odd[k]}, 3, 0});
}

// Rectangular cross-only plan: every 256 x 256 block of the [2 M_a] x [2 M_b] rectangle, column-block major.
void build_groups_rect(int Na, int Nb, int P, std::vector<xtc::PairGroup>& g) {
    g.clear();
    const int Ra = (2 * Na * P + xtc::kPairRows - 1) / xtc::kPairRows;
    const int Rb = (2 * Nb * P + xtc::kPairRows - 1) / xtc::kPairRows;
    for (int cb = 0; cb < Rb; ++cb)
        for (int rb = 0; rb < Ra; ++rb) {
            const xtc::PairTile t{rb * xtc::kPairRows, cb * xtc::kPairRows};
            g.push_back(xtc::PairGroup{{t, t}, 0, 0});
        }
}

int resolve_kernel(const corr_plan* h) {
    if (!h->tma_ok) return CORR_KERNEL_SIMT;
    if (h->kernel != CORR_KERNEL_AUTO) return h->kernel;
    if (h->Nb) return h->max_clusters[0] > 0 ? CORR_KERNEL_PAIR : CORR_KERNEL_SIMT;
    // CORR_KERNEL_QUAD (multicast between two pairs) is never chosen: measured 12 % slower than PAIR at config 4
    // (profiles/): the multicast saves L2 reads but not delivered bytes, and couples the two pairs' pipelines.
    // PAIR vs SINGLE by executed MACs per sample and channel: a pair MAC costs ~0.72 of a 1-CTA MAC (half the operand
    // bytes from L2), but 256 x 256 tiles pad ragged 2M far more than 128-row tiles do.  Measured crossover (T = 2048,
    // N = 72 .. 384): PAIR wins iff pair MACs / single MACs < 1.39.
    if (h->max_clusters[0] <= 0 || 2 * h->M < 256) return CORR_KERNEL_SINGLE;
    double single_macs = 0.0;
    for (const xtc::TileDesc& t : h->h_tiles) single_macs += static_cast<double>(xtc::kTileRows) * t.ncols;
    const double pair_macs = static_cast<double>(h->h_groups[0].size()) * xtc::kPairRows * xtc::kTileCols;
    return pair_macs < 1.39 * single_macs ? CORR_KERNEL_PAIR : CORR_KERNEL_SINGLE;
}

size_t input_bytes(const corr_plan* h) {
    return static_cast<size_t>(h->T) * h->C * h->M * h->sample_bytes;
}
size_t output_bytes(const corr_plan* h) {
    return static_cast<size_t>(h->C) * h->B * h->P * h->P * 8;
}
size_t workspace_bytes(const corr_plan* h) {
    return 2 * static_cast<size_t>(h->C) * h->M * h->Tp * h->sample_bytes;
}

int encode_map(corr_plan* h, CUtensorMap* map, const void* ptr, int M, int box_rows) {
    const int elt = h->sample_bytes / 2;                       // bytes per real component
    const cuuint64_t W = static_cast<cuuint64_t>(h->C) * 2 * M;
    cuuint64_t dims[2] = {W, static_cast<cuuint64_t>(h->T)};
    cuuint64_t strides[1] = {W * elt};
    cuuint32_t box[2] = {static_cast<cuuint32_t>(128 / elt), static_cast<cuuint32_t>(box_rows)};
    cuuint32_t estr[2] = {1, 1};
    const CUresult r = h->encode(map, elt == 1 ? CU_TENSOR_MAP_DATA_TYPE_UINT8 : CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 2,
                                 const_cast<void*>(ptr), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                 CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                                 CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(h, CORR_ECUDA, "cuTensorMapEncodeTiled failed with CUresult %d", static_cast<int>(r));
    return CORR_OK;
}

// Pair kernels: `ptr` viewed as [n_dump][T / n_dump][C*2M] (rank 3), box [128 B][stage samples][1]: a box never crosses
// from one integration into the next, rows past an integration's end are zero-filled.
int encode_map3(corr_plan* h, CUtensorMap* map, const void* ptr, int M, int box_rows, int n_dump) {
    const int elt = h->sample_bytes / 2;
    const cuuint64_t W = static_cast<cuuint64_t>(h->C) * 2 * M;
    const cuuint64_t Ts = static_cast<cuuint64_t>(h->T / n_dump);
    cuuint64_t dims[3] = {W, Ts, static_cast<cuuint64_t>(n_dump)};
    cuuint64_t strides[2] = {W * elt, Ts * W * elt};
    cuuint32_t box[3] = {static_cast<cuuint32_t>(128 / elt), static_cast<cuuint32_t>(box_rows), 1};
    cuuint32_t estr[3] = {1, 1, 1};
    const CUresult r = h->encode(map, elt == 1 ? CU_TENSOR_MAP_DATA_TYPE_UINT8 : CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 3,
                                 const_cast<void*>(ptr), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                 CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                                 CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(h, CORR_ECUDA, "cuTensorMapEncodeTiled (rank 3) failed with CUresult %d", static_cast<int>(r));
    return CORR_OK;
}

// Tensor maps of `in` viewed as [T][C*2M]: box [128 B][stage samples] for the 1-CTA kernel and for the pair kernels.
int encode_input_map(corr_plan* h, const void* in, int n_dump = 1) {
    if (h->tmap_in_ptr == in && h->tmap_dumps == n_dump) return CORR_OK;
    h->tmap_in_ptr = nullptr;
    const int elt = h->sample_bytes / 2;
    int rc = encode_map(h, &h->tmap_in, in, h->M, elt == 1 ? xtc::Cfg<1>::kKStage : xtc::Cfg<2>::kKStage);
    if (rc == CORR_OK)
        rc = encode_map3(h, &h->tmap_pair, in, h->M, (elt == 1 ? xtc::kPairStageK<1> : xtc::kPairStageK<2>) / xtc::kPairBoxes, n_dump);
    if (rc == CORR_OK) { h->tmap_in_ptr = in; h->tmap_dumps = n_dump; }
    return rc;
}

int encode_input_map_b(corr_plan* h, const void* in_b) {
    if (h->tmap_b_ptr == in_b) return CORR_OK;
    h->tmap_b_ptr = nullptr;
    h->tmap_dumps = 1;
    const int elt = h->sample_bytes / 2;
    const int rc = encode_map3(h, &h->tmap_b, in_b, h->Mb, (elt == 1 ? xtc::kPairStageK<1> : xtc::kPairStageK<2>) / xtc::kPairBoxes, 1);
    if (rc == CORR_OK) h->tmap_b_ptr = in_b;
    return rc;
}

int launch_direct(corr_plan* h, const void* in, void* out, int accumulate, cudaStream_t st) {
    int rc = encode_input_map(h, in);
    if (rc != CORR_OK) return rc;
    xtc::Params prm;
    prm.tiles = h->d_tiles;
    prm.tiles_per_chan = static_cast<int>(h->h_tiles.size());
    prm.n_tiles = static_cast<long long>(h->h_tiles.size()) * h->C;
    prm.n_station = h->N;
    prm.n_pol = h->P;
    prm.n_chan = h->C;
    prm.n_time = h->T;
    prm.M = h->M;
    prm.n_baseline = h->B;
    prm.n_station_b = 0;
    prm.M_b = 0;
    prm.n_dump = 1;
    prm.out = out;
    prm.accumulate = accumulate ? 1 : 0;
    // samples per TMEM accumulation pass: everything for int32 (exact); 1024 for fp32 (see xengine_tc.cuh)
    prm.k_chunk = h->dtype == CORR_CI8 ? (1 << 30) : xtc::kFloatChunk;      // int32 sums are exact: one pass
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
        xtc::xengine_direct_kernel<1><<<static_cast<unsigned>(grid), xtc::kNumThreads, xtc::kSmemBytes, st>>>(h->tmap_in, prm);
    else
        xtc::xengine_direct_kernel<2><<<static_cast<unsigned>(grid), xtc::kNumThreads, xtc::kSmemBytes, st>>>(h->tmap_in, prm);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail_cuda(h, e, "xengine_direct_kernel launch");
    h->last_launches += 1;
    return CORR_OK;
}

template <int kElt, int kPairs>
cudaError_t launch_pair_kernel(const CUtensorMap& tmap, const CUtensorMap& tmap_b, const xtc::PairParams& pp, unsigned clusters,
                               cudaStream_t st) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(clusters * 2 * kPairs);
    cfg.blockDim = dim3(xtc::kNumThreads);
    cfg.dynamicSmemBytes = xtc::kPairSmemBytes;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = 2 * kPairs;
    at[0].val.clusterDim.y = 1;
    at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, xtc::xengine_pair_kernel<kElt, kPairs>, tmap, tmap_b, pp);
}

int launch_pair(corr_plan* h, const void* in, const void* in_b, void* out, int accumulate, cudaStream_t st,
                int pairs_per_cluster, int n_dump = 1) {
    int rc = encode_input_map(h, in, n_dump);
    if (rc == CORR_OK && h->Nb) rc = encode_input_map_b(h, in_b);
    if (rc != CORR_OK) return rc;
    const CUtensorMap& map_b = h->Nb ? h->tmap_b : h->tmap_pair;
    const int v = pairs_per_cluster - 1;
    xtc::PairParams pp;
    pp.base.tiles = nullptr;
    pp.base.tiles_per_chan = 0;
    pp.base.n_tiles = 0;
    pp.base.n_station = h->N;
    pp.base.n_pol = h->P;
    pp.base.n_chan = h->C;
    pp.base.n_time = h->T / n_dump;
    pp.base.n_dump = n_dump;
    pp.base.M = h->M;
    pp.base.n_baseline = h->B;
    pp.base.n_station_b = h->Nb;
    pp.base.M_b = h->Mb;
    pp.base.out = out;
    pp.base.accumulate = accumulate ? 1 : 0;
    pp.base.k_chunk = h->dtype == CORR_CI8 ? (1 << 30) : xtc::kFloatChunk;      // int32 sums are exact: one pass
#ifdef CORR_STATS
    static unsigned long long* d_stats = nullptr;
    if (!d_stats) cudaMalloc(&d_stats, 8 * 160 * sizeof(unsigned long long));
    cudaMemsetAsync(d_stats, 0, 8 * 160 * sizeof(unsigned long long), st);
    pp.base.stats = d_stats;
#endif
    pp.groups = h->d_groups[v];
    pp.groups_per_chan = static_cast<int>(h->h_groups[v].size());
    pp.n_groups = static_cast<long long>(pp.groups_per_chan) * h->C * n_dump;
    const unsigned clusters = static_cast<unsigned>(pp.n_groups < h->max_clusters[v] ? pp.n_groups : h->max_clusters[v]);
    if (pp.n_groups > (1ll << 31) - 4096) return fail(h, CORR_EINVAL, "xengine_pair_kernel: %lld tiles exceed the tile feed's range", pp.n_groups);
    pp.sched_counter = h->d_sched + (h->sched_seq++ % kSchedRing);
    cudaError_t e = cudaMemsetAsync(pp.sched_counter, 0, sizeof(unsigned int), st);
    if (e != cudaSuccess) return fail_cuda(h, e, "tile-feed counter reset");
    if (h->dtype == CORR_CI8)
        e = v ? launch_pair_kernel<1, 2>(h->tmap_pair, map_b, pp, clusters, st) : launch_pair_kernel<1, 1>(h->tmap_pair, map_b, pp, clusters, st);
    else
        e = v ? launch_pair_kernel<2, 2>(h->tmap_pair, map_b, pp, clusters, st) : launch_pair_kernel<2, 1>(h->tmap_pair, map_b, pp, clusters, st);
    if (e != cudaSuccess) return fail_cuda(h, e, "xengine_pair_kernel launch");
#ifdef CORR_STATS
    if (getenv("CORR_STATS_PRINT")) {
        static unsigned long long hs[8 * 160];
        cudaStreamSynchronize(st);
        cudaMemcpy(hs, d_stats, sizeof(hs), cudaMemcpyDeviceToHost);
        const int nb = static_cast<int>(clusters) * 2 * pairs_per_cluster;
        double a[8] = {0};
        for (int b = 0; b < nb; ++b) for (int k = 0; k < 8; ++k) a[k] += static_cast<double>(hs[b * 8 + k]) / nb;
        double lead_tempty = 0, lead_full = 0;
        for (int b = 0; b < nb; b += 2) { lead_tempty += hs[b * 8 + 2] / (nb / 2.0); lead_full += hs[b * 8 + 3] / (nb / 2.0); }
        double tmin = 1e30, tmax = 0;
        for (int b = 0; b < nb; ++b) { if (hs[b * 8] < tmin) tmin = hs[b * 8]; if (hs[b * 8] > tmax) tmax = hs[b * 8]; }
        fprintf(stderr, "[corr stats] producer loop clk: min %.0f max %.0f (spread %.1f %%)\n", tmin, tmax, 100.0 * (tmax - tmin) / tmax);
        fprintf(stderr, "[corr stats] clk/CTA: total %.0f | producer wait empty %.0f | mma wait tmem-empty %.0f, wait full %.0f | epi(warp2) wait tmem-full %.0f, drain %.0f\n",
                a[0], a[1], lead_tempty, lead_full, a[4], a[5]);
    }
#endif
    h->last_launches += 1;
    return CORR_OK;
}

int launch_simt(corr_plan* h, const void* in, const void* in_b, void* out, int accumulate, cudaStream_t st) {
    xsimt::Params prm;
    prm.in = in;
    prm.in_b = in_b;
    prm.n_station_b = h->Nb;
    prm.out = out;
    prm.n_station = h->N;
    prm.n_pol = h->P;
    prm.n_chan = h->C;
    prm.n_time = h->T;
    prm.n_baseline = h->B;
    prm.n_vis = static_cast<long long>(h->C) * h->B * h->P * h->P;
    prm.accumulate = accumulate ? 1 : 0;
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

int launch_corner_turn(corr_plan* h, const void* in, void* ws, cudaStream_t st) {
    cturn::Params prm;
    prm.in = in;
    prm.ws = ws;
    prm.ws_rot = static_cast<uint8_t*>(ws) + workspace_bytes(h) / 2;
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
    } else if (kernel == CORR_KERNEL_PAIR || kernel == CORR_KERNEL_QUAD) {
        std::vector<xtc::PairGroup> g;
        build_groups(n_station, n_pol, kernel == CORR_KERNEL_QUAD ? 2 : 1, g);
        for (const xtc::PairGroup& x : g)
            for (int k = 0; k < (kernel == CORR_KERNEL_QUAD ? 2 : 1); ++k) {
                flat.push_back(x.t[k].row0);
                flat.push_back(x.t[k].col0);
                flat.push_back(k == 1 && x.share == 3 ? 0 : xtc::kTileCols);     // 0: duplicate, computed but not written
            }
    } else {
        return CORR_EINVAL;
    }
    const int n = static_cast<int>(flat.size() / 3);
    for (int k = 0; k < n && k < max_tiles; ++k)
        for (int q = 0; q < 3; ++q) tiles3[3 * k + q] = flat[3 * k + q];
    return n;
}

static corr_handle create_plan(int n_station, int n_station_b, int n_pol, int n_chan, int n_time, int dtype) {
    g_create_error[0] = 0;
    if (!valid_geometry(n_station, n_pol, dtype) || n_station_b < 0 || n_chan < 1 || n_time < 1) {
        fail(nullptr, CORR_EINVAL, "corr_create: invalid geometry N=%d Nb=%d P=%d C=%d T=%d dtype=%d", n_station, n_station_b,
             n_pol, n_chan, n_time, dtype);
        return nullptr;
    }
    const long long M = static_cast<long long>(n_station) * n_pol;
    const long long Mb = static_cast<long long>(n_station_b) * n_pol;
    const long long W = static_cast<long long>(n_chan) * 2 * (M > Mb ? M : Mb);
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
    if (prop.major != 10) {
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
    h->tmap_b_ptr = nullptr;
    h->t_total = 0;
    h->last_launches = 0;
    h->d_tiles = nullptr;
    h->kernel = CORR_KERNEL_AUTO;
    h->d_groups[0] = h->d_groups[1] = nullptr;
    h->d_sched = nullptr;
    h->sched_seq = 0;
    h->max_clusters[0] = h->max_clusters[1] = 0;
    h->encode = nullptr;
    h->tmap_in_ptr = nullptr;
    h->Tp = (n_time + 63) / 64 * 64;
    h->d_in_stage = nullptr;
    h->d_out_stage = nullptr;
    h->own_stream = nullptr;
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
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult qres;
        e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
        if (e != cudaSuccess || qres != cudaDriverEntryPointSuccess || !fn) {
            fail(nullptr, CORR_ECUDA, "corr_create: cuTensorMapEncodeTiled entry point unavailable (%s)",
                 cudaGetErrorString(e));
            corr_destroy(h);
            return nullptr;
        }
        h->encode = reinterpret_cast<EncodeTiledFn>(fn);
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
        // CTA-pair kernels: group tables and the number of co-resident clusters (the persistent grid)
        for (int v = 0; v < (h->Nb ? 1 : 2) && e == cudaSuccess; ++v) {
            if (h->Nb) build_groups_rect(h->N, h->Nb, h->P, h->h_groups[v]);
            else build_groups(h->N, h->P, v + 1, h->h_groups[v]);
            const size_t bytes = h->h_groups[v].size() * sizeof(xtc::PairGroup);
            e = cudaMalloc(&h->d_groups[v], bytes);
            if (e == cudaSuccess) e = cudaMemcpy(h->d_groups[v], h->h_groups[v].data(), bytes, cudaMemcpyHostToDevice);
            const void* fn_ptr = h->dtype == CORR_CI8
                                     ? (v ? (const void*)xtc::xengine_pair_kernel<1, 2> : (const void*)xtc::xengine_pair_kernel<1, 1>)
                                     : (v ? (const void*)xtc::xengine_pair_kernel<2, 2> : (const void*)xtc::xengine_pair_kernel<2, 1>);
            if (e == cudaSuccess) e = cudaFuncSetAttribute(fn_ptr, cudaFuncAttributeMaxDynamicSharedMemorySize, xtc::kPairSmemBytes);
            if (e == cudaSuccess) {
                cudaLaunchConfig_t cfg = {};
                cfg.gridDim = dim3(static_cast<unsigned>(h->sm_count / (2 * (v + 1)) * (2 * (v + 1))));
                cfg.blockDim = dim3(xtc::kNumThreads);
                cfg.dynamicSmemBytes = xtc::kPairSmemBytes;
                cudaLaunchAttribute at[1];
                at[0].id = cudaLaunchAttributeClusterDimension;
                at[0].val.clusterDim.x = 2 * (v + 1);
                at[0].val.clusterDim.y = 1;
                at[0].val.clusterDim.z = 1;
                cfg.attrs = at;
                cfg.numAttrs = 1;
                int n = 0;
                if (cudaOccupancyMaxActiveClusters(&n, fn_ptr, &cfg) == cudaSuccess) h->max_clusters[v] = n;
                else cudaGetLastError();          // pair kernels unavailable: resolve_kernel falls back
            }
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
    return create_plan(n_station, 0, n_pol, n_chan, n_time, dtype);
}

corr_handle corr_create_cross(int n_station_a, int n_station_b, int n_pol, int n_chan, int n_time, int dtype) {
    if (n_station_b < 1) {
        g_create_error[0] = 0;
        fail(nullptr, CORR_EINVAL, "corr_create_cross: invalid geometry Na=%d Nb=%d", n_station_a, n_station_b);
        return nullptr;
    }
    return create_plan(n_station_a, n_station_b, n_pol, n_chan, n_time, dtype);
}

void corr_destroy(corr_handle h) {
    if (!h) return;
    if (h->d_tiles) cudaFree(h->d_tiles);
    if (h->d_sched) cudaFree(h->d_sched);
    if (h->d_groups[0]) cudaFree(h->d_groups[0]);
    if (h->d_groups[1]) cudaFree(h->d_groups[1]);
    if (h->d_in_stage) cudaFree(h->d_in_stage);
    if (h->d_out_stage) cudaFree(h->d_out_stage);
    if (h->own_stream) cudaStreamDestroy(h->own_stream);
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
    if (h->Nb && (kernel == CORR_KERNEL_SINGLE || kernel == CORR_KERNEL_QUAD))
        return fail(h, CORR_EUNSUPPORTED, "corr_set_kernel: cross plans run on the PAIR or the SIMT kernel");
    if ((kernel == CORR_KERNEL_PAIR && h->max_clusters[0] <= 0) || (kernel == CORR_KERNEL_QUAD && h->max_clusters[1] <= 0))
        return fail(h, CORR_EUNSUPPORTED, "corr_set_kernel: no co-resident clusters for kernel %d on this device", kernel);
    h->kernel = kernel;
    return CORR_OK;
}
int corr_last_launch_count(corr_handle h) { return h ? h->last_launches : CORR_EINVAL; }

static int run_fengine(const void* in, void* out, int n_stream, long long n_spectra, bool int8_out, float scale, void* stream) {
    g_create_error[0] = 0;
    if (!in || !out || n_stream < 1 || n_spectra < 1 || n_spectra > 0x7fffffffLL || (int8_out && !(scale > 0.0f)))
        return fail(nullptr, CORR_EINVAL, "corr_fengine: invalid arguments (n_stream=%d, n_spectra=%lld)", n_stream, n_spectra);
    if ((reinterpret_cast<uintptr_t>(in) & 15) || (reinterpret_cast<uintptr_t>(out) & (int8_out ? 1 : 3)))
        return fail(nullptr, CORR_EINVAL, "corr_fengine: `in` must be 16-byte and `out` element aligned");
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

int corr_corner_turn(corr_handle h, const void* in, void* ws, void* stream) {
    if (!h) return CORR_EINVAL;
    if (h->Nb) return fail(h, CORR_EINVAL, "corr_corner_turn: not available on cross plans");
    if (!in || !ws) return fail(h, CORR_EINVAL, "corr_corner_turn: NULL pointer");
    if ((reinterpret_cast<uintptr_t>(in) & 15) || (reinterpret_cast<uintptr_t>(ws) & 127))
        return fail(h, CORR_EINVAL, "corr_corner_turn: `in` must be 16-byte and `ws` 128-byte aligned");
    if (!h->tma_ok)
        return fail(h, CORR_EUNSUPPORTED, "corr_corner_turn: per-channel row of %lld B is not a multiple of 16",
                    static_cast<long long>(h->M) * h->sample_bytes);
    h->last_launches = 0;
    return launch_corner_turn(h, in, ws, static_cast<cudaStream_t>(stream));
}

static int run_xengine(corr_handle h, const void* in, const void* in_b, void* out, int accumulate, void* stream);

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
    h->last_launches = 0;
    h->t_total = Ts;
    const int kernel = resolve_kernel(h);
    if (kernel != CORR_KERNEL_SIMT && h->max_clusters[0] > 0)
        return launch_pair(h, in, nullptr, out, 0, st, 1, n_dump);       // any TMA-addressable geometry runs on the pair kernel
    // SIMT: one launch per integration on slices of `in` and `out`
    const int T_full = h->T;
    int rc = CORR_OK;
    h->T = Ts;
    for (int d = 0; d < n_dump && rc == CORR_OK; ++d)
        rc = launch_simt(h, static_cast<const uint8_t*>(in) + d * input_bytes(h), nullptr,
                         static_cast<uint8_t*>(out) + d * output_bytes(h), 0, st);
    h->T = T_full;
    return rc;
}

int corr_xengine_cross(corr_handle h, const void* in_a, const void* in_b, void* out, int accumulate, void* stream) {
    if (!h) return CORR_EINVAL;
    if (!h->Nb) return fail(h, CORR_EINVAL, "corr_xengine_cross: this is not a cross plan; call corr_xengine");
    if (!in_b || (reinterpret_cast<uintptr_t>(in_b) & 15))
        return fail(h, CORR_EINVAL, "corr_xengine_cross: `in_b` must be a non-NULL, 16-byte aligned device pointer");
    return run_xengine(h, in_a, in_b, out, accumulate, stream);
}

static int run_xengine(corr_handle h, const void* in, const void* in_b, void* out, int accumulate, void* stream) {
    if (!in || !out) return fail(h, CORR_EINVAL, "corr_xengine: NULL pointer");
    if ((reinterpret_cast<uintptr_t>(in) & 15) || (reinterpret_cast<uintptr_t>(out) & 15))
        return fail(h, CORR_EINVAL, "corr_xengine: `in` and `out` must be 16-byte aligned");
    const long long t_next = accumulate ? h->t_total + h->T : h->T;
    if (h->dtype == CORR_CI8 && t_next > kMaxIntegrationCi8)
        return fail(h, CORR_EOVERFLOW, "corr_xengine: integrating %lld samples would overflow int32 (limit %lld)", t_next,
                    kMaxIntegrationCi8);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    h->last_launches = 0;
    int rc;
    switch (resolve_kernel(h)) {
        case CORR_KERNEL_QUAD: rc = launch_pair(h, in, in_b, out, accumulate, st, 2); break;
        case CORR_KERNEL_PAIR: rc = launch_pair(h, in, in_b, out, accumulate, st, 1); break;
        case CORR_KERNEL_SINGLE: rc = launch_direct(h, in, out, accumulate, st); break;
        default: rc = launch_simt(h, in, in_b, out, accumulate, st); break;
    }
    if (rc == CORR_OK) h->t_total = t_next;
    return rc;
}

int corr_xengine_host(corr_handle h, const void* in_host, void* out_host, int accumulate) {
    if (!h) return CORR_EINVAL;
    if (h->Nb) return fail(h, CORR_EINVAL, "corr_xengine_host: not available on cross plans");
    if (!in_host) return fail(h, CORR_EINVAL, "corr_xengine_host: NULL input pointer");
    cudaError_t e;
    if (!h->own_stream) {
        e = cudaStreamCreateWithFlags(&h->own_stream, cudaStreamNonBlocking);
        if (e != cudaSuccess) return fail_cuda(h, e, "cudaStreamCreate");
    }
    if (!h->d_in_stage) {
        e = cudaMalloc(&h->d_in_stage, input_bytes(h));
        if (e != cudaSuccess) return fail(h, CORR_ENOMEM, "corr_xengine_host: input staging: %s", cudaGetErrorString(e));
    }
    if (!h->d_out_stage) {
        if (accumulate) return fail(h, CORR_EINVAL, "corr_xengine_host: accumulate without a previous call");
        e = cudaMalloc(&h->d_out_stage, output_bytes(h));
        if (e != cudaSuccess) return fail(h, CORR_ENOMEM, "corr_xengine_host: output staging: %s", cudaGetErrorString(e));
    }
    e = cudaMemcpyAsync(h->d_in_stage, in_host, input_bytes(h), cudaMemcpyHostToDevice, h->own_stream);
    if (e != cudaSuccess) return fail_cuda(h, e, "H2D copy");
    const int rc = corr_xengine(h, h->d_in_stage, h->d_out_stage, accumulate, h->own_stream);
    if (rc != CORR_OK) return rc;
    if (out_host) {
        e = cudaMemcpyAsync(out_host, h->d_out_stage, output_bytes(h), cudaMemcpyDeviceToHost, h->own_stream);
        if (e != cudaSuccess) return fail_cuda(h, e, "D2H copy");
    }
    e = cudaStreamSynchronize(h->own_stream);
    if (e != cudaSuccess) return fail_cuda(h, e, "corr_xengine_host: stream synchronize");
    return CORR_OK;
}

}  // extern "C"
