// k_noalloc.cu - mwa_grid_visibilities_noalloc: the tile-owned register gridder (K3c, k_gather.cu) with its binning
// workspace in a file-scope device array instead of a plan's cudaMalloc'ed workspace.
//
// For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid
// it): the entry point takes no plan and calls no cudaMalloc, cudaFree or allocating library routine, ever.  The
// kernels are the ones the plan path runs (scale_kernel, the binning kernels of k_bin.cu, gather_kernel); only where
// their scratch lives differs.  The scratch is g_noalloc_scratch below: kNoallocBytes (about 7.6 MB) of every GPU that
// loads this library, held until the process exits.  That fixes the maximum sizes of a call (MWA_GRID_NOALLOC_MAX_* in
// include/mwa_grid.h): larger calls are rejected with MWA_GRID_ERR_INVALID.
//
// In host code `g_noalloc_scratch` is a host-side stand-in for the symbol, NOT a device address; the device address is
// taken once per device, with that device current, by cudaGetSymbolAddress (noalloc_device_state) and only that
// pointer is handed to the launchers.
//
// All calls on one device share the array and it keeps the contents of the call before: the binning step clears the
// parts that must start at zero (the counters and block states in `misc` and the bucket histogram - launch_binning's
// two cudaMemsetAsync - everything else is fully overwritten before it is read).  Two calls that overlap on the GPU
// (different streams without an ordering between them, or two host threads) race on the array: order them.
#include <cmath>
#include <cstdint>
#include <mutex>
#include <string>

#include "../../include/mwa_grid.h"
#include "plan.h"

namespace mwa {

constexpr long long kNoallocMaxVis = MWA_GRID_NOALLOC_MAX_VIS;
constexpr int kNoallocMaxChan = MWA_GRID_NOALLOC_MAX_CHAN;
constexpr int kNoallocMaxGridN = MWA_GRID_NOALLOC_MAX_GRID_N;

constexpr size_t round256(size_t n) { return (n + 255) & ~size_t(255); }

// layout of the scratch array: every section starts on a 256-byte boundary
constexpr int kNaBuckets = ((kNoallocMaxGridN + kBucketCells - 1) / kBucketCells) * ((kNoallocMaxGridN + kBucketCells - 1) / kBucketCells);
constexpr int kNaTiles = ((kNoallocMaxGridN + kTile - 1) / kTile) * ((kNoallocMaxGridN + kTile - 1) / kTile);
constexpr size_t kOffScale = 0;                                                               // double [max_chan]
constexpr size_t kOffGroup = kOffScale + round256(sizeof(double) * kNoallocMaxChan);           // double [max_chan / 32][4]
constexpr size_t kOffScaleRef = kOffGroup + round256(sizeof(double) * 4 * ((kNoallocMaxChan + 31) / 32));   // double [1]
constexpr size_t kOffDispatch = kOffScaleRef + 256;                                           // int [1]
constexpr size_t kOffMisc = kOffDispatch + 256;                                               // int [kMiscInts]
constexpr size_t kOffBucketCount = kOffMisc + round256(sizeof(int) * kMiscInts);              // int [buckets + 1]
constexpr size_t kOffBucketCursor = kOffBucketCount + round256(sizeof(int) * (kNaBuckets + 1));   // int [buckets]
constexpr size_t kOffTileOrder = kOffBucketCursor + round256(sizeof(int) * kNaBuckets);       // int [tiles]
constexpr size_t kOffTileWeight = kOffTileOrder + round256(sizeof(int) * kNaTiles);           // int [tiles]
constexpr size_t kOffPerm = kOffTileWeight + round256(sizeof(int) * kNaTiles);                // int [max_vis]
constexpr size_t kOffPermTmp = kOffPerm + round256(sizeof(int) * kNoallocMaxVis);             // int [max_vis]
constexpr size_t kOffUvSorted = kOffPermTmp + round256(sizeof(int) * kNoallocMaxVis);         // double2 [max_vis]
constexpr size_t kOffRowSorted = kOffUvSorted + round256(sizeof(double2) * kNoallocMaxVis);   // double4 [max_vis]
constexpr size_t kNoallocBytes = kOffRowSorted + round256(sizeof(double) * 4 * kNoallocMaxVis);
static_assert(kNoallocBytes <= (size_t)8 << 20, "the static scratch is meant to stay modest (<= 8 MiB)");

static __device__ __align__(256) unsigned char g_noalloc_scratch[kNoallocBytes];

// per device: the device address of the array on that device and the SM count, resolved on the first call there
constexpr int kNaMaxDevices = 64;
struct NoallocDevice {
    unsigned char* base = nullptr;
    int sm_count = 0;
};
static NoallocDevice g_na_dev[kNaMaxDevices];
static std::mutex g_na_mutex;

static bool noalloc_device_state(int dev, NoallocDevice* out) {
    if (dev < 0 || dev >= kNaMaxDevices) { set_error("device ordinal out of range for the no-allocation entry point"); return false; }
    std::lock_guard<std::mutex> lock(g_na_mutex);
    NoallocDevice& d = g_na_dev[dev];
    if (!d.base) {
        // `dev` is the current device (the caller asked cudaGetDevice): the symbol resolves to this device's copy
        unsigned char* ptr = nullptr;
        if (!cuda_ok(cudaGetSymbolAddress((void**)&ptr, g_noalloc_scratch), "cudaGetSymbolAddress(noalloc scratch)")) return false;
        if (!ptr || (reinterpret_cast<uintptr_t>(ptr) & 255) != 0) { set_error("noalloc scratch: bad device address"); return false; }
        int sms = 0;
        if (!cuda_ok(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev), "sm count")) return false;
        d.sm_count = sms;
        d.base = ptr;
    }
    *out = d;
    return true;
}

static bool na_aligned(const void* p, size_t a) { return (reinterpret_cast<uintptr_t>(p) % a) == 0; }

}  // namespace mwa

using namespace mwa;

extern "C" int mwa_grid_visibilities_noalloc(int grid_n, double cell_du, int support_W, int oversample_O,
                                             const float* kernel_table_dev, const double* uv_f64, const double* freqs,
                                             const float* vis_c64, const float* weights, long long n_vis, int n_chan,
                                             float* grid_out, void* stream) {
    set_error("");
    // the checks of mwa_grid_plan_create and mwa_grid_visibilities, then the limits of the static scratch
    if (grid_n < 16 || (grid_n & 1)) { set_error("grid_n must be even and >= 16"); return MWA_GRID_ERR_INVALID; }
    if (support_W < 1 || support_W > 15 || !(support_W & 1)) { set_error("support_W must be odd and in [1, 15]"); return MWA_GRID_ERR_INVALID; }
    if (grid_n < 2 * support_W) { set_error("grid_n must be >= 2 * support_W"); return MWA_GRID_ERR_INVALID; }
    if (oversample_O < 2 || oversample_O > 64 || (oversample_O & 1)) { set_error("oversample_O must be even and in [2, 64]"); return MWA_GRID_ERR_INVALID; }
    if (!(cell_du > 0.0) || !std::isfinite(cell_du)) { set_error("cell_du must be finite and > 0"); return MWA_GRID_ERR_INVALID; }
    if (n_vis < 0 || n_chan < 0) { set_error("n_vis and n_chan must be >= 0"); return MWA_GRID_ERR_INVALID; }
    if (grid_n > kNoallocMaxGridN) {
        set_error("mwa_grid_visibilities_noalloc: grid_n " + std::to_string(grid_n) + " exceeds the static scratch (MWA_GRID_NOALLOC_MAX_GRID_N = " +
                  std::to_string(kNoallocMaxGridN) + "); use a plan");
        return MWA_GRID_ERR_INVALID;
    }
    if (n_vis > kNoallocMaxVis) {
        set_error("mwa_grid_visibilities_noalloc: n_vis " + std::to_string(n_vis) + " exceeds the static scratch (MWA_GRID_NOALLOC_MAX_VIS = " +
                  std::to_string(kNoallocMaxVis) + "); use a plan or split the rows with accumulate-into");
        return MWA_GRID_ERR_INVALID;
    }
    if (n_chan > kNoallocMaxChan) {
        set_error("mwa_grid_visibilities_noalloc: n_chan " + std::to_string(n_chan) + " exceeds the static scratch (MWA_GRID_NOALLOC_MAX_CHAN = " +
                  std::to_string(kNoallocMaxChan) + "); use a plan or split the channels");
        return MWA_GRID_ERR_INVALID;
    }
    if (n_chan == 0) return MWA_GRID_OK;
    if (!kernel_table_dev) { set_error("kernel_table_dev is NULL"); return MWA_GRID_ERR_INVALID; }
    if (!freqs) { set_error("freqs is NULL"); return MWA_GRID_ERR_INVALID; }
    if (!grid_out) { set_error("grid_out is NULL"); return MWA_GRID_ERR_INVALID; }
    if (n_vis > 0 && (!uv_f64 || !vis_c64)) { set_error("uv_f64 / vis_c64 is NULL"); return MWA_GRID_ERR_INVALID; }
    if (!na_aligned(uv_f64, 16) || !na_aligned(freqs, 8) || !na_aligned(vis_c64, 32) || !na_aligned(weights, 4) ||
        !na_aligned(grid_out, 16) || !na_aligned(kernel_table_dev, 4)) {
        set_error("alignment: uv_f64 16 bytes, freqs 8, vis_c64 32, weights 4, grid_out 16, kernel_table_dev 4");
        return MWA_GRID_ERR_INVALID;
    }

    int dev = -1;
    if (!cuda_ok(cudaGetDevice(&dev), "cudaGetDevice")) return MWA_GRID_ERR_CUDA;
    NoallocDevice nd;
    if (!noalloc_device_state(dev, &nd)) return MWA_GRID_ERR_CUDA;

    // a plan on the stack whose workspace pointers are sections of the static array: the launchers of the plan path run
    // unchanged.  Nothing in it is owned (no destroy), nothing is allocated.
    Plan p;
    p.geom.N = grid_n;
    p.geom.W = support_W;
    p.geom.h = (support_W - 1) / 2;
    p.geom.O = oversample_O;
    p.geom.o_shift = -1;
    for (int k = 1; k <= 6; ++k)
        if ((1 << k) == oversample_O) p.geom.o_shift = k;
    p.geom.inv_du = 1.0 / cell_du;
    p.cell_du = cell_du;
    p.d_table = const_cast<float*>(kernel_table_dev);   // read only by the kernels
    p.design = MWA_GRID_DESIGN_GATHER;
    p.device = dev;
    p.sm_count = nd.sm_count;
    Workspace& ws = p.ws;
    unsigned char* b = nd.base;
    ws.d_scale = reinterpret_cast<double*>(b + kOffScale);
    ws.d_group = reinterpret_cast<double*>(b + kOffGroup);
    ws.cap_chan = kNoallocMaxChan;
    ws.d_scale_ref = reinterpret_cast<double*>(b + kOffScaleRef);
    ws.d_dispatch = reinterpret_cast<int*>(b + kOffDispatch);
    ws.d_misc = reinterpret_cast<int*>(b + kOffMisc);
    ws.d_bucket_count = reinterpret_cast<int*>(b + kOffBucketCount);
    ws.d_bucket_cursor = reinterpret_cast<int*>(b + kOffBucketCursor);
    ws.cap_buckets = kNaBuckets;
    ws.d_tile_order = reinterpret_cast<int*>(b + kOffTileOrder);
    ws.d_tile_weight = reinterpret_cast<int*>(b + kOffTileWeight);
    ws.cap_tiles = kNaTiles;
    ws.d_perm = reinterpret_cast<int*>(b + kOffPerm);
    ws.d_perm_tmp = reinterpret_cast<int*>(b + kOffPermTmp);
    ws.d_uv_sorted = reinterpret_cast<double2*>(b + kOffUvSorted);
    ws.d_row_sorted = reinterpret_cast<double*>(b + kOffRowSorted);
    ws.cap_vis = kNoallocMaxVis;

    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    if (n_vis == 0) {                                        // R10: every cell is written
        if (!cuda_ok(cudaMemsetAsync(grid_out, 0, (size_t)n_chan * 4 * grid_n * grid_n * 8, st), "memset grid")) return MWA_GRID_ERR_CUDA;
        return MWA_GRID_OK;
    }
    if (!launch_scale(&p, freqs, n_chan, st)) return MWA_GRID_ERR_CUDA;
    if (!launch_binning(&p, uv_f64, n_vis, n_chan, st)) return MWA_GRID_ERR_CUDA;          // clears misc and the histogram
    if (!launch_gather(&p, vis_c64, weights, n_vis, n_chan, grid_out, nullptr, st)) return MWA_GRID_ERR_CUDA;
    return MWA_GRID_OK;
}
