// plan.h - the plan object behind the C ABI and the launchers of the individual kernels.
#pragma once
#include <cuda_runtime.h>
#include <new>
#include <string>
#include "index.cuh"

namespace mwa {

// Binning geometry (a3).  Rows are sorted once per call by the bucket of their position at the TOP
// frequency of the call (largest extent); every channel's position is a radial contraction of that one.
constexpr int kBucketCells = 8;     // bucket side in cells at the reference scale
constexpr int kChanMinChannels = 8; // AUTO picks a channel-SIMD kernel (K6 / K5) only from this many channels on
constexpr int kTile = 16;           // gridding tile side in cells (one warp owns one tile of one channel)
// d_misc (ints, zeroed by every call's binning step): [0..3] work counters, [4..11] diagnostics, [12..13] hit-list pool
// cursor (u64), [14..15] K6 item counts, [16..] tile-weight histogram (4096), then the block states of chan_order_kernel
constexpr int kWeightBins = 1024;            // tile-weight histogram bins (weight clipped to kWeightBins - 1), heaviest first
#ifndef MWA_HEAVY_TILE_WEIGHT
#define MWA_HEAVY_TILE_WEIGHT 256
#endif
constexpr int kHeavyTileWeight = MWA_HEAVY_TILE_WEIGHT;        // a tile with this many rows in the buckets under it (~ 480 hits with the halo) is "heavy":
                                             // K3c grids its items with the four warps of a CTA when items are few (k_gather.cu)
constexpr int kMiscHeavyTiles = 16 + kWeightBins - 1 - kHeavyTileWeight;   // after tile_order_scatter_kernel: end of that weight bin
                                             // in tile_order = the number of tiles at least that heavy
constexpr int kMiscHeavyCounter = 16 + kWeightBins;   // [1] work counter of K3c's heavy items
constexpr int kMiscHeavyStat = 2048 + 46;              // long long: heavy items of the last K3c call (last_stats()[31])
constexpr int kMiscTailStart = 16 + 4080;    // [1] first entry of the last channel group in K6's list of items with hits
constexpr int kMiscOrderState = 16 + 4096;
constexpr int kMiscScanState = kMiscOrderState + 2048;   // block states of bin_scan_kernel (<= 1024 blocks: 4 M buckets)
constexpr int kMiscBigList = kMiscScanState + 1024;    // [0] number of big buckets of bin_order_kernel, [1..1023] their ids
constexpr int kMiscInts = kMiscBigList + 1024;

struct Workspace {
    // a1
    double* d_scale = nullptr;       // [n_chan]
    double* d_group = nullptr;       // [ceil(n_chan / 32)][4] per channel group: s_lo, s_hi, s_ref/s_lo, s_ref/s_hi
    int cap_chan = 0;
    // a3
    double* d_scale_ref = nullptr;   // [1] max over channels of s_c
    int* d_bucket_count = nullptr;   // [nb*nb + 1] histogram, then exclusive scan = bucket_start
    int* d_bucket_cursor = nullptr;  // [nb*nb] scatter cursors
    int cap_buckets = 0;
    int* d_perm = nullptr;           // [n_vis] row ids sorted by bucket, ascending inside a bucket
    int* d_perm_tmp = nullptr;       // [n_vis] scatter target before the in-bucket ordering
    double2* d_uv_sorted = nullptr;  // [n_vis] uv of the sorted rows
    double* d_row_sorted = nullptr;  // [n_vis][4] (u, v, row id, 0) of the sorted rows: one 32 B record per row (K5)
    long long cap_vis = 0;
    int* d_tile_order = nullptr;     // [n_tiles] tile ids, heaviest first
    int* d_tile_weight = nullptr;    // [n_tiles]
    int* d_misc = nullptr;           // small counters
    int* d_dispatch = nullptr;       // [1] design picked on the device for AUTO: 0 = gather (K3c), 1 = chan (K6 / K5)
    int cap_tiles = 0;
    // K6 (k_chanws.cu) pre-pass outputs
    unsigned* d_pre = nullptr;       // [n_vis][ceil(n_chan / 32) * 32] packed exact indices, by row
    void* d_bb = nullptr;            // [ceil(n_chan / 32)][n_vis] ushort4 bounding boxes, by sorted position
    size_t cap_pre = 0;              // capacity in (row, padded channel) elements
    int* d_list_cnt = nullptr;       // [n_items] hits per (tile, channel group) item; -1 = not listed
    unsigned* d_list_off = nullptr;  // [n_items] first entry of the item's list in the pool
    void* d_c_desc = nullptr;        // [n_items] int4 (item, hits, list offset, 0) of the items with hits, in item order
    unsigned* d_z_list = nullptr;    // [n_items] the items nothing reaches, in item order
    long long cap_items = 0;         // items the four arrays above are sized for
    void* d_lists = nullptr;         // [pool_cap] uint2 (row, mask): pool of hit lists
    unsigned pool_cap = 0;           // entries in the pool (what this call may use)
    size_t cap_pool = 0;             // entries allocated
    // host-buffer entry point staging
    void* d_stage = nullptr;
    size_t cap_stage = 0;
};

struct Plan {
    GridGeom geom{};
    double cell_du = 0.0;
    float* d_table = nullptr;        // [(O+1)][W] as given
    float* h_table = nullptr;        // host copy
    float* d_table2d = nullptr;      // f3: general 2-D complex table [(O+1)][(O+1)][W][W][2] (plans of mwa_grid_plan_create_2d), else null
    int design = 0;
    int device = 0;
    int sm_count = 148;
    Workspace ws;
    // profiling
    bool profiling = false;
    cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
    bool ev_valid = false;
    int last_launches = 0;
    // f1 imaging step (k_image.cu)
    float* d_inv_corr = nullptr;     // [N] 1 / c^(p' - N/2)
    double* h_corr = nullptr;        // [N] c^(p' - N/2), host copy (fp64)
    int fft_handle[2] = {0, 0};      // cached cuFFT plans ...
    int fft_batch[2] = {0, 0};       // ... and the batch sizes they were made for (0 = none)
    cudaStream_t copy_stream[2] = {nullptr, nullptr};   // host entry point: upload / download streams of the channel-chunk pipeline
    bool mfs = false;                // f3: all channels of a call are summed onto ONE grid [4][N][N] (mwa_grid_plan_set_mfs)
    bool accumulate = false;         // f3: grid_out += instead of = (mwa_grid_plan_set_accumulate)
    long long pool_limit = 0;        // diagnostics: cap on K6's hit-list pool in entries (0 = default sizing)
    bool last_chanws = false;        // AUTO: the channel-SIMD kernel enqueued by the last call was K6 (else K5)
    bool pdl_next = false;           // the kernel enqueued last was the fused pre-pass of a small call (it releases its dependents
                                     // at once): launch_gather, if it comes next, launches with programmatic stream serialisation
};

// ---- programmatic dependent launch (the kernels of one call's pre-pass chain)
// A kernel launched with launch_dependent may become resident while the kernel before it on the stream still runs; it
// must execute pdl_wait() before it touches anything that kernel (or any kernel before that) writes - every kernel of a
// chain does so first thing, in every thread, so completion is transitive - and pdl_release() lets the next kernel of
// the chain become resident in turn.  Both are no-ops in a kernel that was launched the plain way.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_release() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

template <typename... KArgs, typename... Args>
inline cudaError_t launch_dependent(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kern, static_cast<KArgs>(args)...);
}

void set_error(const std::string& msg);
bool cuda_ok(cudaError_t e, const char* what);

// launchers (each returns false after set_error on failure and adds its launches to plan->last_launches)
bool launch_scale(Plan* p, const double* freqs, int n_chan, cudaStream_t st);
bool launch_weights_grid(Plan* p, const double* uv, const float* w, long long n_vis, int n_chan, float* wgrid, cudaStream_t st);
bool launch_count_dropped(Plan* p, const double* uv, long long n_vis, int n_chan, unsigned long long* d_count, cudaStream_t st);
bool launch_indices(Plan* p, const double* uv, long long n_vis, int n_chan, int* out_idx, cudaStream_t st);
bool launch_atomic(Plan* p, const double* uv, const float* vis, const float* w, long long n_vis, int n_chan,
                   float* grid, cudaStream_t st);
bool launch_binning(Plan* p, const double* uv, long long n_vis, int n_chan, cudaStream_t st, bool cleared = false);
bool launch_binning_clear(Plan* p, cudaStream_t st);       // the memsets of launch_binning, to be enqueued before launch_scale (then cleared = true)
bool binning_is_small(const Plan* p, long long n_vis);     // the call's a1 + a3 fit one CTA: launch_small_prepass replaces
bool launch_small_prepass(Plan* p, const double* uv, const double* freqs, long long n_vis, int n_chan, cudaStream_t st);   // launch_scale + launch_binning
bool launch_gather(Plan* p, const float* vis, const float* w, long long n_vis, int n_chan, float* grid,
                   const int* dispatch, cudaStream_t st);
bool probe_fp32(Plan* p, double* tflops_ffma, double* tflops_ffma2, cudaStream_t st);
bool probe_smem_atomics(Plan* p, double* lane_atomics_per_s, cudaStream_t st);
bool chan_supported(const Plan* p, int n_chan);
bool launch_chan(Plan* p, const float* vis, const float* w, long long n_vis, int n_chan, float* grid,
                 const int* dispatch, cudaStream_t st);
bool chanws_supported(const Plan* p, int n_chan);
long long chanws_items(const Plan* p, int n_chan);
bool launch_chanws(Plan* p, const float* vis, const float* w, long long n_vis, int n_chan, float* grid,
                   const int* dispatch, cudaStream_t st);
bool launch_smem(Plan* p, const float* vis, const float* w, long long n_vis, int n_chan, float* grid,
                 cudaStream_t st);
bool launch_image(Plan* p, const float* grid, float* image, long long n_planes, cudaStream_t st);
const double* image_correction_host(Plan* p, cudaStream_t st);
bool launch_stokes(Plan* p, const float* image, const float* matrix, float* out, int n_chan, cudaStream_t st);
void image_release(Plan* p);
bool launch_gather2d(Plan* p, const float* vis, const float* w, long long n_vis, int n_chan, float* grid, cudaStream_t st);
bool launch_romein(Plan* p, const double* uv, const float* vis, const float* w, long long n_vis, int n_chan, float* grid,
                   const int* perm, cudaStream_t st);

}  // namespace mwa
