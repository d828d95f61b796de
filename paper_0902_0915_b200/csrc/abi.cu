// abi.cu - the extern "C" boundary declared in include/mwa_grid.h: argument checks, workspace, dispatch.
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/mwa_grid.h"
#include "plan.h"

namespace mwa {

static thread_local std::string g_last_error;

void set_error(const std::string& msg) { g_last_error = msg; }

bool cuda_ok(cudaError_t e, const char* what) {
    if (e == cudaSuccess) return true;
    set_error(std::string(what) + ": " + cudaGetErrorName(e) + " - " + cudaGetErrorString(e));
    return false;
}

// Grows one workspace array: the new buffer is allocated first and swapped in on success, so a failed call leaves the
// old (smaller) buffer and its capacity valid.
template <typename T>
static bool ensure(T*& ptr, size_t count, const char* what) {
    T* fresh = nullptr;
    if (count > 0) {
        cudaError_t e = cudaMalloc((void**)&fresh, count * sizeof(T));
        if (e != cudaSuccess) {
            cudaGetLastError();
            set_error(std::string("workspace allocation failed (") + what + "): " + cudaGetErrorString(e));
            return false;
        }
    }
    if (ptr) cudaFree(ptr);
    ptr = fresh;
    return true;
}

// returns 0 / MWA_GRID_ERR_NOMEM
static int ensure_workspace(Plan* p, long long n_vis, int n_chan) {
    Workspace& ws = p->ws;
    // every capacity is dropped before its arrays are regrown and restored only when all of them succeeded, so a
    // call after a failed one reallocates instead of running on a partly grown workspace
    if (n_chan > ws.cap_chan) {
        ws.cap_chan = 0;
        if (!ensure(ws.d_scale, (size_t)n_chan, "scale")) return MWA_GRID_ERR_NOMEM;
        if (!ensure(ws.d_group, (size_t)((n_chan + 31) / 32) * 4, "group")) return MWA_GRID_ERR_NOMEM;
        ws.cap_chan = n_chan;
    }
    if (!ws.d_scale_ref && !ensure(ws.d_scale_ref, 1, "scale_ref")) return MWA_GRID_ERR_NOMEM;
    if (!ws.d_dispatch && !ensure(ws.d_dispatch, 1, "dispatch")) return MWA_GRID_ERR_NOMEM;
    const int nb = (p->geom.N + kBucketCells - 1) / kBucketCells;
    const int n_buckets = nb * nb;
    if (n_buckets > ws.cap_buckets) {
        ws.cap_buckets = 0;
        if (!ensure(ws.d_bucket_count, (size_t)n_buckets + 1, "bucket_count")) return MWA_GRID_ERR_NOMEM;
        if (!ensure(ws.d_bucket_cursor, (size_t)n_buckets, "bucket_cursor")) return MWA_GRID_ERR_NOMEM;
        ws.cap_buckets = n_buckets;
    }
    if (n_vis > ws.cap_vis) {
        ws.cap_vis = 0;
        if (!ensure(ws.d_perm, (size_t)n_vis, "perm")) return MWA_GRID_ERR_NOMEM;
        if (!ensure(ws.d_perm_tmp, (size_t)n_vis, "perm_tmp")) return MWA_GRID_ERR_NOMEM;
        if (!ensure(ws.d_uv_sorted, (size_t)n_vis, "uv_sorted")) return MWA_GRID_ERR_NOMEM;
        if (!ensure(ws.d_row_sorted, (size_t)n_vis * 4, "row_sorted")) return MWA_GRID_ERR_NOMEM;
        ws.cap_vis = n_vis;
    }
    const int nt = (p->geom.N + kTile - 1) / kTile;
    const int n_tiles = nt * nt;
    if (n_tiles > ws.cap_tiles) {
        ws.cap_tiles = 0;
        if (!ensure(ws.d_tile_order, (size_t)n_tiles, "tile_order")) return MWA_GRID_ERR_NOMEM;
        if (!ensure(ws.d_tile_weight, (size_t)n_tiles, "tile_weight")) return MWA_GRID_ERR_NOMEM;
        ws.cap_tiles = n_tiles;
    }
    if (!ws.d_misc && !ensure(ws.d_misc, (size_t)kMiscInts, "misc")) return MWA_GRID_ERR_NOMEM;
    const bool want_ws = (p->design == MWA_GRID_DESIGN_CHANWS || (p->design == MWA_GRID_DESIGN_AUTO && n_chan >= kChanMinChannels)) &&
                         chanws_supported(p, n_chan);
    const size_t n_pre = want_ws ? (size_t)n_vis * (size_t)((n_chan + 31) / 32) * 32 : 0;
    if (n_pre > ws.cap_pre) {
        ws.cap_pre = 0;
        if (!ensure(ws.d_pre, n_pre, "packed indices")) return MWA_GRID_ERR_NOMEM;
        unsigned long long* bb = (unsigned long long*)ws.d_bb;
        if (!ensure(bb, n_pre / 32, "bounding boxes")) { ws.d_bb = bb; return MWA_GRID_ERR_NOMEM; }
        ws.d_bb = bb;
        ws.cap_pre = n_pre;
    }
    if (want_ws) {
        // hit lists of K6: per item a count and an offset into a pool sized for 12 candidate entries per (row, channel
        // group) - about 1.5 x what the slot reservation of chan_list_kernel asks for on C4 - capped at 1 GiB; an item
        // that finds the pool full is swept inside the gridding kernel instead, so the size is never a correctness matter
        const long long items = chanws_items(p, n_chan);
        if (items > ws.cap_items) {
            ws.cap_items = 0;
            if (!ensure(ws.d_list_cnt, (size_t)items, "hit counts")) return MWA_GRID_ERR_NOMEM;
            if (!ensure(ws.d_list_off, (size_t)items, "hit list offsets")) return MWA_GRID_ERR_NOMEM;
            if (!ensure(ws.d_z_list, (size_t)items + 16, "zero item list")) return MWA_GRID_ERR_NOMEM;   // read 16 at a time
            int4* cd = (int4*)ws.d_c_desc;
            if (!ensure(cd, (size_t)items, "item descriptors")) { ws.d_c_desc = cd; return MWA_GRID_ERR_NOMEM; }
            ws.d_c_desc = cd;
            ws.cap_items = items;
        }
        long long pool = n_vis * (long long)((n_chan + 31) / 32) * 12;
        if (pool > (1LL << 27)) pool = 1LL << 27;
        if (pool < 1024) pool = 1024;
        if (p->pool_limit > 0 && pool > p->pool_limit) pool = p->pool_limit;
        if ((size_t)pool > ws.cap_pool) {
            ws.cap_pool = 0;
            unsigned long long* l = (unsigned long long*)ws.d_lists;
            if (!ensure(l, (size_t)pool, "hit lists")) { ws.d_lists = l; return MWA_GRID_ERR_NOMEM; }
            ws.d_lists = l;
            ws.cap_pool = (size_t)pool;
        }
        ws.pool_cap = (unsigned)pool;
    }
    return MWA_GRID_OK;
}

static bool aligned(const void* p, size_t a) { return (reinterpret_cast<uintptr_t>(p) % a) == 0; }

static int check_common(Plan* p, const double* uv, const double* freqs, long long n_vis, int n_chan, bool device_pointers = true) {
    if (!p) { set_error("plan is NULL"); return MWA_GRID_ERR_INVALID; }
    if (n_vis < 0 || n_chan < 0) { set_error("n_vis and n_chan must be >= 0"); return MWA_GRID_ERR_INVALID; }
    if (n_vis > 0x7fffffffLL) { set_error("n_vis must fit in 31 bits"); return MWA_GRID_ERR_INVALID; }
    if (n_chan > 0 && !freqs) { set_error("freqs is NULL"); return MWA_GRID_ERR_INVALID; }
    if (n_vis > 0 && n_chan > 0 && !uv) { set_error("uv_f64 is NULL"); return MWA_GRID_ERR_INVALID; }
    if (device_pointers) {                        // the kernels read uv as double2; host buffers are only copied
        if (!aligned(uv, 16)) { set_error("uv_f64 must be 16-byte aligned"); return MWA_GRID_ERR_INVALID; }
        if (!aligned(freqs, 8)) { set_error("freqs must be 8-byte aligned"); return MWA_GRID_ERR_INVALID; }
    }
    return MWA_GRID_OK;
}


static int grid_device(Plan* p, const double* uv, const double* freqs, const float* vis, const float* weights,
                       long long n_vis, int n_chan, float* grid, cudaStream_t st) {
    p->last_launches = 0;
    p->pdl_next = false;
    if (n_chan == 0) return MWA_GRID_OK;
    int dev = -1;
    if (!cuda_ok(cudaGetDevice(&dev), "cudaGetDevice")) return MWA_GRID_ERR_CUDA;
    if (dev != p->device) {                       // the workspace and the kernel attributes live on the plan's device
        set_error("the current CUDA device (" + std::to_string(dev) + ") is not the device the plan was created on (" +
                  std::to_string(p->device) + ")");
        return MWA_GRID_ERR_INVALID;
    }
    int rc = ensure_workspace(p, n_vis, n_chan);
    if (rc != MWA_GRID_OK) return rc;
    const bool prof = p->profiling;
    if (prof) {
        for (auto& e : p->ev)
            if (!e && !cuda_ok(cudaEventCreate(&e), "cudaEventCreate")) return MWA_GRID_ERR_CUDA;
        cudaEventRecord(p->ev[0], st);
    }
    const int design = p->design;
    const bool bins = design != MWA_GRID_DESIGN_ATOMIC && design != MWA_GRID_DESIGN_ROMEIN && n_vis > 0;
    if (bins && binning_is_small(p, n_vis)) {              // launch-bound calls: a1 + a3 in one launch
        if (!launch_small_prepass(p, uv, freqs, n_vis, n_chan, st)) return MWA_GRID_ERR_CUDA;
    } else {
        // the memsets of the binning step go first, so that its first kernel can follow scale_kernel as a dependent launch
        if (bins && !launch_binning_clear(p, st)) return MWA_GRID_ERR_CUDA;
        if (!launch_scale(p, freqs, n_chan, st)) return MWA_GRID_ERR_CUDA;
        if (bins && !launch_binning(p, uv, n_vis, n_chan, st, true)) return MWA_GRID_ERR_CUDA;
    }
    {
        // the pre-pass kernels form a chain of programmatic dependent launches; only a gather kernel that DIRECTLY follows
        // the chain joins it (nothing may sit between the two: no stage timer, no memset of the MFS grid, no other kernel)
        const bool direct = !prof && !p->d_table2d && (design == MWA_GRID_DESIGN_GATHER ||
                                                      (design == MWA_GRID_DESIGN_AUTO && (n_chan < kChanMinChannels || p->mfs)));
        p->pdl_next = p->pdl_next && direct && !(p->mfs && !p->accumulate);
#ifdef MWA_NO_PDL
        p->pdl_next = false;                                     // A/B measurement build only
#endif
    }
    if (prof) cudaEventRecord(p->ev[1], st);
    bool ok = false;
    const int out_chan = p->mfs ? 1 : n_chan;              // grids the call writes
    if (n_vis == 0 && p->accumulate) {
        ok = true;                                // nothing to add
    } else if (n_vis == 0) {
        ok = cuda_ok(cudaMemsetAsync(grid, 0, (size_t)out_chan * 4 * p->geom.N * p->geom.N * 8, st), "memset grid");
        p->last_launches += 1;
    } else {
        if (p->mfs && design != MWA_GRID_DESIGN_AUTO && design != MWA_GRID_DESIGN_GATHER && design != MWA_GRID_DESIGN_ATOMIC &&
            design != MWA_GRID_DESIGN_ROMEIN && design != MWA_GRID_DESIGN_ROMEIN_SORTED) {
            set_error("multi-frequency synthesis is implemented by the designs AUTO (= GATHER), GATHER, ATOMIC and ROMEIN only");
            return MWA_GRID_ERR_INVALID;
        }
        if (p->accumulate && (design == MWA_GRID_DESIGN_SMEM || design == MWA_GRID_DESIGN_CHAN)) {
            set_error("accumulate-into is implemented by the designs AUTO, GATHER, CHANWS, ATOMIC and ROMEIN only");
            return MWA_GRID_ERR_INVALID;
        }
        if (p->d_table2d) {                           // plans of mwa_grid_plan_create_2d: one kernel (k_gather2d.cu)
            if ((design != MWA_GRID_DESIGN_AUTO && design != MWA_GRID_DESIGN_GATHER) || p->accumulate || p->mfs) {
                set_error("a plan with a 2-D kernel table grids with the design AUTO / GATHER only, without accumulate-into or MFS");
                return MWA_GRID_ERR_INVALID;
            }
            ok = launch_gather2d(p, vis, weights, n_vis, n_chan, grid, st);
        } else
        switch (design) {
            case MWA_GRID_DESIGN_ATOMIC: ok = launch_atomic(p, uv, vis, weights, n_vis, n_chan, grid, st); break;
            case MWA_GRID_DESIGN_SMEM: ok = launch_smem(p, vis, weights, n_vis, n_chan, grid, st); break;
            case MWA_GRID_DESIGN_ROMEIN: ok = launch_romein(p, uv, vis, weights, n_vis, n_chan, grid, nullptr, st); break;
            case MWA_GRID_DESIGN_ROMEIN_SORTED: ok = launch_romein(p, uv, vis, weights, n_vis, n_chan, grid, p->ws.d_perm, st); break;
            case MWA_GRID_DESIGN_GATHER: ok = launch_gather(p, vis, weights, n_vis, n_chan, grid, nullptr, st); break;
            case MWA_GRID_DESIGN_CHAN: ok = launch_chan(p, vis, weights, n_vis, n_chan, grid, nullptr, st); break;
            case MWA_GRID_DESIGN_CHANWS: ok = launch_chanws(p, vis, weights, n_vis, n_chan, grid, nullptr, st); break;
            case MWA_GRID_DESIGN_AUTO:
                // the choice is made on the device by scale_kernel (the host never reads freqs): both kernels
                // are enqueued and the one that was not picked returns at once
                ok = true;
                if (n_chan < kChanMinChannels || p->mfs) {
                    // the device-side rule can only pick the gather kernel: the channel-SIMD kernels and their pre-passes
                    // are not enqueued at all (small single-channel calls are launch-bound)
                    p->last_chanws = false;
                    ok = launch_gather(p, vis, weights, n_vis, n_chan, grid, nullptr, st);
                    break;
                }
                p->last_chanws = chanws_supported(p, n_chan);
                if (p->last_chanws) ok = launch_chanws(p, vis, weights, n_vis, n_chan, grid, p->ws.d_dispatch, st);
                else if (chan_supported(p, n_chan) && !p->accumulate) ok = launch_chan(p, vis, weights, n_vis, n_chan, grid, p->ws.d_dispatch, st);
                ok = ok && launch_gather(p, vis, weights, n_vis, n_chan, grid, p->ws.d_dispatch, st);
                break;
            default: set_error("unknown design"); return MWA_GRID_ERR_INVALID;
        }
    }
    if (!ok) return MWA_GRID_ERR_CUDA;
    if (prof) {
        cudaEventRecord(p->ev[2], st);
        p->ev_valid = true;
    }
    return MWA_GRID_OK;
}

}  // namespace mwa

using namespace mwa;

extern "C" {

const char* mwa_grid_last_error(void) { return g_last_error.c_str(); }

static mwa_grid_plan* plan_create_common(int grid_n, double cell_du, int support_W, int oversample_O, const float* kernel_table,
                                         bool two_d) {
    g_last_error.clear();
    if (grid_n < 16 || grid_n > 16384 || (grid_n & 1)) { set_error("grid_n must be even and in [16, 16384]"); return nullptr; }
    if (support_W < 1 || support_W > 15 || !(support_W & 1)) { set_error("support_W must be odd and in [1, 15]"); return nullptr; }
    if (grid_n < 2 * support_W) { set_error("grid_n must be >= 2 * support_W"); return nullptr; }
    if (oversample_O < 2 || oversample_O > 64 || (oversample_O & 1)) { set_error("oversample_O must be even and in [2, 64]"); return nullptr; }
    if (two_d && oversample_O > 62) { set_error("2-D tables: oversample_O must be <= 62"); return nullptr; }
    if (!(cell_du > 0.0) || !std::isfinite(cell_du)) { set_error("cell_du must be finite and > 0"); return nullptr; }
    if (!kernel_table) { set_error("kernel_table is NULL"); return nullptr; }
    Plan* p = new (std::nothrow) Plan();
    if (!p) { set_error("out of host memory"); return nullptr; }
    p->geom.N = grid_n;
    p->geom.W = support_W;
    p->geom.h = (support_W - 1) / 2;
    p->geom.O = oversample_O;
    p->geom.o_shift = -1;
    for (int k = 1; k <= 6; ++k)
        if ((1 << k) == oversample_O) p->geom.o_shift = k;
    p->geom.inv_du = 1.0 / cell_du;
    p->cell_du = cell_du;
    const size_t O1 = (size_t)oversample_O + 1;
    const size_t n = two_d ? O1 * O1 * support_W * support_W * 2 : O1 * support_W;
    float** d_dst = two_d ? &p->d_table2d : &p->d_table;
    if (!two_d) {
        p->h_table = new (std::nothrow) float[n];
        if (!p->h_table) { set_error("out of host memory"); delete p; return nullptr; }
        std::memcpy(p->h_table, kernel_table, n * sizeof(float));
    }
    if (!cuda_ok(cudaGetDevice(&p->device), "cudaGetDevice") ||
        !cuda_ok(cudaDeviceGetAttribute(&p->sm_count, cudaDevAttrMultiProcessorCount, p->device), "sm count") ||
        !cuda_ok(cudaMalloc((void**)d_dst, n * sizeof(float)), "cudaMalloc table") ||
        !cuda_ok(cudaMemcpy(*d_dst, kernel_table, n * sizeof(float), cudaMemcpyHostToDevice), "copy table")) {
        mwa_grid_plan_destroy(reinterpret_cast<mwa_grid_plan*>(p));
        return nullptr;
    }
    return reinterpret_cast<mwa_grid_plan*>(p);
}

mwa_grid_plan* mwa_grid_plan_create(int grid_n, double cell_du, int support_W, int oversample_O,
                                    const float* kernel_table) {
    return plan_create_common(grid_n, cell_du, support_W, oversample_O, kernel_table, false);
}

mwa_grid_plan* mwa_grid_plan_create_2d(int grid_n, double cell_du, int support_W, int oversample_O,
                                       const float* kernel_table_2d) {
    return plan_create_common(grid_n, cell_du, support_W, oversample_O, kernel_table_2d, true);
}

void mwa_grid_plan_destroy(mwa_grid_plan* plan) {
    if (!plan) return;
    Plan* p = reinterpret_cast<Plan*>(plan);
    Workspace& ws = p->ws;
    void* ptrs[] = {p->d_table, p->d_table2d, ws.d_scale, ws.d_group, ws.d_scale_ref, ws.d_bucket_count, ws.d_bucket_cursor, ws.d_perm, ws.d_perm_tmp,
                    ws.d_uv_sorted, ws.d_row_sorted, ws.d_tile_order, ws.d_tile_weight, ws.d_misc, ws.d_dispatch, ws.d_stage,
                    ws.d_pre, ws.d_bb, ws.d_list_cnt, ws.d_list_off, ws.d_c_desc, ws.d_z_list, ws.d_lists};
    for (void* q : ptrs)
        if (q) cudaFree(q);
    image_release(p);
    for (auto& cs : p->copy_stream)
        if (cs) cudaStreamDestroy(cs);
    for (auto& e : p->ev)
        if (e) cudaEventDestroy(e);
    delete[] p->h_table;
    delete p;
}

int mwa_image_from_grid(mwa_grid_plan* plan, const float* grid, float* image, long long n_planes, void* stream) {
    g_last_error.clear();
    Plan* p = reinterpret_cast<Plan*>(plan);
    if (!p) { set_error("plan is NULL"); return MWA_GRID_ERR_INVALID; }
    if (!p->d_table) { set_error("the convolution correction is defined for separable 1-D tables only"); return MWA_GRID_ERR_INVALID; }
    if (n_planes < 0) { set_error("n_planes must be >= 0"); return MWA_GRID_ERR_INVALID; }
    p->last_launches = 0;
    if (n_planes == 0) return MWA_GRID_OK;
    if (!grid || !image || !aligned(grid, 16) || !aligned(image, 16)) { set_error("grid and image must be non-NULL and 16-byte aligned"); return MWA_GRID_ERR_INVALID; }
    if (grid != image) {
        const size_t bytes = (size_t)n_planes * p->geom.N * p->geom.N * 8;
        const char *a = (const char*)grid, *b = (const char*)image;
        if (a < b + bytes && b < a + bytes) { set_error("grid and image must be the same buffer or not overlap"); return MWA_GRID_ERR_INVALID; }
    }
    int dev = -1;
    if (!cuda_ok(cudaGetDevice(&dev), "cudaGetDevice")) return MWA_GRID_ERR_CUDA;
    if (dev != p->device) { set_error("the current CUDA device is not the device the plan was created on"); return MWA_GRID_ERR_INVALID; }
    return launch_image(p, grid, image, n_planes, reinterpret_cast<cudaStream_t>(stream)) ? MWA_GRID_OK : MWA_GRID_ERR_CUDA;
}

int mwa_image_stokes(mwa_grid_plan* plan, const float* image, const float* matrix, float* stokes_out, int n_chan, void* stream) {
    g_last_error.clear();
    Plan* p = reinterpret_cast<Plan*>(plan);
    if (!p) { set_error("plan is NULL"); return MWA_GRID_ERR_INVALID; }
    if (n_chan < 0) { set_error("n_chan must be >= 0"); return MWA_GRID_ERR_INVALID; }
    p->last_launches = 0;
    if (n_chan == 0) return MWA_GRID_OK;
    if (!image || !matrix || !stokes_out || !aligned(image, 8) || !aligned(stokes_out, 8) || !aligned(matrix, 16)) {
        set_error("image, matrix and stokes_out must be non-NULL; image / stokes_out 8-byte, matrix 16-byte aligned");
        return MWA_GRID_ERR_INVALID;
    }
    if (image != stokes_out) {
        const size_t bytes = (size_t)n_chan * 4 * p->geom.N * p->geom.N * 8;
        const char *a = (const char*)image, *b = (const char*)stokes_out;
        if (a < b + bytes && b < a + bytes) { set_error("image and stokes_out must be the same buffer or not overlap"); return MWA_GRID_ERR_INVALID; }
    }
    int dev = -1;
    if (!cuda_ok(cudaGetDevice(&dev), "cudaGetDevice")) return MWA_GRID_ERR_CUDA;
    if (dev != p->device) { set_error("the current CUDA device is not the device the plan was created on"); return MWA_GRID_ERR_INVALID; }
    return launch_stokes(p, image, matrix, stokes_out, n_chan, reinterpret_cast<cudaStream_t>(stream)) ? MWA_GRID_OK : MWA_GRID_ERR_CUDA;
}

int mwa_image_correction(mwa_grid_plan* plan, double* out_corr, int n) {
    g_last_error.clear();
    Plan* p = reinterpret_cast<Plan*>(plan);
    if (!p || !out_corr || n < 0) { set_error("bad argument"); return MWA_GRID_ERR_INVALID; }
    if (!p->d_table) { set_error("the convolution correction is defined for separable 1-D tables only"); return MWA_GRID_ERR_INVALID; }
    const double* c = image_correction_host(p, nullptr);
    if (!c) return MWA_GRID_ERR_CUDA;
    const int k = n < p->geom.N ? n : p->geom.N;
    std::memcpy(out_corr, c, (size_t)k * sizeof(double));
    return k;
}

int mwa_grid_plan_set_design(mwa_grid_plan* plan, int design) {
    if (!plan) { set_error("plan is NULL"); return MWA_GRID_ERR_INVALID; }
    if (design < MWA_GRID_DESIGN_AUTO || design > MWA_GRID_DESIGN_ROMEIN_SORTED) { set_error("unknown design"); return MWA_GRID_ERR_INVALID; }
    reinterpret_cast<Plan*>(plan)->design = design;
    return MWA_GRID_OK;
}

int mwa_grid_plan_set_accumulate(mwa_grid_plan* plan, int enabled) {
    if (!plan) { set_error("plan is NULL"); return MWA_GRID_ERR_INVALID; }
    reinterpret_cast<Plan*>(plan)->accumulate = enabled != 0;
    return MWA_GRID_OK;
}

int mwa_grid_plan_set_mfs(mwa_grid_plan* plan, int enabled) {
    if (!plan) { set_error("plan is NULL"); return MWA_GRID_ERR_INVALID; }
    reinterpret_cast<Plan*>(plan)->mfs = enabled != 0;
    return MWA_GRID_OK;
}

int mwa_grid_plan_set_profiling(mwa_grid_plan* plan, int enabled) {
    if (!plan) { set_error("plan is NULL"); return MWA_GRID_ERR_INVALID; }
    Plan* p = reinterpret_cast<Plan*>(plan);
    p->profiling = enabled != 0;
    p->ev_valid = false;
    return MWA_GRID_OK;
}

int mwa_grid_plan_stage_ms(mwa_grid_plan* plan, float* out_ms, int n) {
    if (!plan || !out_ms || n < 0) { set_error("bad argument"); return MWA_GRID_ERR_INVALID; }
    Plan* p = reinterpret_cast<Plan*>(plan);
    if (!p->ev_valid) { set_error("no profiled call recorded"); return MWA_GRID_ERR_INVALID; }
    if (!cuda_ok(cudaEventSynchronize(p->ev[2]), "cudaEventSynchronize")) return MWA_GRID_ERR_CUDA;
    float v[3] = {0, 0, 0};
    cudaEventElapsedTime(&v[0], p->ev[0], p->ev[1]);
    cudaEventElapsedTime(&v[1], p->ev[1], p->ev[2]);
    cudaEventElapsedTime(&v[2], p->ev[0], p->ev[2]);
    int k = n < 3 ? n : 3;
    for (int i = 0; i < k; ++i) out_ms[i] = v[i];
    return k;
}

int mwa_grid_probe_fp32(mwa_grid_plan* plan, double* out_tflops, void* stream) {
    if (!plan || !out_tflops) { set_error("bad argument"); return MWA_GRID_ERR_INVALID; }
    return probe_fp32(reinterpret_cast<Plan*>(plan), &out_tflops[0], &out_tflops[1], reinterpret_cast<cudaStream_t>(stream))
               ? MWA_GRID_OK : MWA_GRID_ERR_CUDA;
}

int mwa_grid_probe_smem_atomics(mwa_grid_plan* plan, double* out_rate, void* stream) {
    if (!plan || !out_rate) { set_error("bad argument"); return MWA_GRID_ERR_INVALID; }
    return probe_smem_atomics(reinterpret_cast<Plan*>(plan), out_rate, reinterpret_cast<cudaStream_t>(stream)) ? MWA_GRID_OK : MWA_GRID_ERR_CUDA;
}


int mwa_grid_plan_set_list_pool(mwa_grid_plan* plan, long long entries) {
    if (!plan || entries < 0) { set_error("bad argument"); return MWA_GRID_ERR_INVALID; }
    reinterpret_cast<Plan*>(plan)->pool_limit = entries;
    return MWA_GRID_OK;
}

int mwa_grid_plan_last_launches(const mwa_grid_plan* plan) {
    return plan ? reinterpret_cast<const Plan*>(plan)->last_launches : 0;
}

int mwa_grid_plan_last_design(mwa_grid_plan* plan) {
    if (!plan) { set_error("plan is NULL"); return MWA_GRID_ERR_INVALID; }
    Plan* p = reinterpret_cast<Plan*>(plan);
    if (p->design != MWA_GRID_DESIGN_AUTO) return p->design;
    if (!p->ws.d_dispatch) { set_error("no gridding call recorded"); return MWA_GRID_ERR_INVALID; }
    int v = 0;
    if (!cuda_ok(cudaMemcpy(&v, p->ws.d_dispatch, sizeof(int), cudaMemcpyDeviceToHost), "read dispatch")) return MWA_GRID_ERR_CUDA;
    if (v != 1) return MWA_GRID_DESIGN_GATHER;
    return p->last_chanws ? MWA_GRID_DESIGN_CHANWS : MWA_GRID_DESIGN_CHAN;
}

int mwa_grid_plan_last_stats(mwa_grid_plan* plan, long long* out, int n) {
    if (!plan || !out || n < 0) { set_error("bad argument"); return MWA_GRID_ERR_INVALID; }
    Plan* p = reinterpret_cast<Plan*>(plan);
    if (!p->ws.d_misc) { set_error("no gridding call recorded"); return MWA_GRID_ERR_INVALID; }
    int v[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    long long t[24];
    if (!cuda_ok(cudaMemcpy(v, p->ws.d_misc + 4, sizeof(v), cudaMemcpyDeviceToHost), "read stats")) return MWA_GRID_ERR_CUDA;
    if (!cuda_ok(cudaMemcpy(t, p->ws.d_misc + 2048, sizeof(t), cudaMemcpyDeviceToHost), "read stats")) return MWA_GRID_ERR_CUDA;
    const int k = n < 32 ? n : 32;
    for (int i = 0; i < k; ++i) out[i] = i < 8 ? (long long)v[i] : t[i - 8];   // [8..31]: phase clocks of a -DK6_TIMING build, else 0
    return k;
}

int mwa_grid_compute_indices(mwa_grid_plan* plan, const double* uv_f64, const double* freqs, long long n_vis,
                             int n_chan, int* out_idx, void* stream) {
    g_last_error.clear();
    Plan* p = reinterpret_cast<Plan*>(plan);
    int rc = check_common(p, uv_f64, freqs, n_vis, n_chan);
    if (rc != MWA_GRID_OK) return rc;
    if (n_vis == 0 || n_chan == 0) return MWA_GRID_OK;
    if (!out_idx || !aligned(out_idx, 16)) { set_error("out_idx must be non-NULL and 16-byte aligned"); return MWA_GRID_ERR_INVALID; }
    rc = ensure_workspace(p, n_vis, n_chan);
    if (rc != MWA_GRID_OK) return rc;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    p->last_launches = 0;
    if (!launch_scale(p, freqs, n_chan, st)) return MWA_GRID_ERR_CUDA;
    if (!launch_indices(p, uv_f64, n_vis, n_chan, out_idx, st)) return MWA_GRID_ERR_CUDA;
    return MWA_GRID_OK;
}

int mwa_grid_weights_grid(mwa_grid_plan* plan, const double* uv_f64, const double* freqs, const float* weights, long long n_vis,
                          int n_chan, float* wgrid_out, void* stream) {
    g_last_error.clear();
    Plan* p = reinterpret_cast<Plan*>(plan);
    int rc = check_common(p, uv_f64, freqs, n_vis, n_chan);
    if (rc != MWA_GRID_OK) return rc;
    if (n_chan == 0) { p->last_launches = 0; return MWA_GRID_OK; }
    if (!p->d_table) { set_error("the weights grid is implemented for separable 1-D tables only"); return MWA_GRID_ERR_INVALID; }
    if (!wgrid_out || !aligned(wgrid_out, 4) || !aligned(weights, 4)) { set_error("wgrid_out must be non-NULL; wgrid_out and weights 4-byte aligned"); return MWA_GRID_ERR_INVALID; }
    rc = ensure_workspace(p, n_vis, n_chan);
    if (rc != MWA_GRID_OK) return rc;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    p->last_launches = 0;
    if (!launch_scale(p, freqs, n_chan, st)) return MWA_GRID_ERR_CUDA;
    return launch_weights_grid(p, uv_f64, weights, n_vis, n_chan, wgrid_out, st) ? MWA_GRID_OK : MWA_GRID_ERR_CUDA;
}

int mwa_grid_count_dropped(mwa_grid_plan* plan, const double* uv_f64, const double* freqs, long long n_vis, int n_chan,
                           long long* out_count, void* stream) {
    g_last_error.clear();
    Plan* p = reinterpret_cast<Plan*>(plan);
    int rc = check_common(p, uv_f64, freqs, n_vis, n_chan);
    if (rc != MWA_GRID_OK) return rc;
    if (!out_count) { set_error("out_count is NULL"); return MWA_GRID_ERR_INVALID; }
    *out_count = 0;
    if (n_vis == 0 || n_chan == 0) return MWA_GRID_OK;
    rc = ensure_workspace(p, n_vis, n_chan);
    if (rc != MWA_GRID_OK) return rc;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    p->last_launches = 0;
    unsigned long long* d_count = reinterpret_cast<unsigned long long*>(p->ws.d_misc + 12);   // the call's scratch counter
    if (!cuda_ok(cudaMemsetAsync(d_count, 0, sizeof(unsigned long long), st), "memset counter")) return MWA_GRID_ERR_CUDA;
    if (!launch_scale(p, freqs, n_chan, st)) return MWA_GRID_ERR_CUDA;
    if (!launch_count_dropped(p, uv_f64, n_vis, n_chan, d_count, st)) return MWA_GRID_ERR_CUDA;
    unsigned long long h = 0;
    if (!cuda_ok(cudaMemcpyAsync(&h, d_count, sizeof(h), cudaMemcpyDeviceToHost, st), "read counter") ||
        !cuda_ok(cudaStreamSynchronize(st), "count_dropped_kernel")) return MWA_GRID_ERR_CUDA;
    *out_count = (long long)h;
    return MWA_GRID_OK;
}

int mwa_grid_visibilities(mwa_grid_plan* plan, const double* uv_f64, const double* freqs, const float* vis_c64,
                          const float* weights, long long n_vis, int n_chan, float* grid_out, void* stream) {
    g_last_error.clear();
    Plan* p = reinterpret_cast<Plan*>(plan);
    int rc = check_common(p, uv_f64, freqs, n_vis, n_chan);
    if (rc != MWA_GRID_OK) return rc;
    if (n_chan == 0) { p->last_launches = 0; return MWA_GRID_OK; }
    if (!grid_out || !aligned(grid_out, 16)) { set_error("grid_out must be non-NULL and 16-byte aligned"); return MWA_GRID_ERR_INVALID; }
    if (n_vis > 0 && (!vis_c64 || !aligned(vis_c64, 32))) { set_error("vis_c64 must be non-NULL and 32-byte aligned"); return MWA_GRID_ERR_INVALID; }
    if (!aligned(weights, 4)) { set_error("weights must be 4-byte aligned"); return MWA_GRID_ERR_INVALID; }
    return grid_device(p, uv_f64, freqs, vis_c64, weights, n_vis, n_chan, grid_out, reinterpret_cast<cudaStream_t>(stream));
}

int mwa_grid_visibilities_host(mwa_grid_plan* plan, const double* uv_f64, const double* freqs, const float* vis_c64,
                               const float* weights, long long n_vis, int n_chan, float* grid_out, void* stream) {
    g_last_error.clear();
    Plan* p = reinterpret_cast<Plan*>(plan);
    int rc = check_common(p, uv_f64, freqs, n_vis, n_chan, false);
    if (rc != MWA_GRID_OK) return rc;
    if (n_chan == 0) { p->last_launches = 0; return MWA_GRID_OK; }
    if (!grid_out) { set_error("grid_out is NULL"); return MWA_GRID_ERR_INVALID; }
    if (n_vis > 0 && !vis_c64) { set_error("vis_c64 is NULL"); return MWA_GRID_ERR_INVALID; }
    if (p->accumulate || p->mfs) { set_error("accumulate-into and multi-frequency synthesis work on device grids only (mwa_grid_visibilities)"); return MWA_GRID_ERR_INVALID; }
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    auto up = [](size_t b) { return (b + 255) & ~size_t(255); };
    // Channels own their grids, so the call is pipelined over channel chunks (multiples of 32 channels, ~8 per call):
    // the upload of chunk k + 1 (copy stream) and the download of chunk k - 1's grids (second copy stream) run under the
    // gridding of chunk k on the caller's stream.  PCIe carries both directions at once; what stays exposed is the first
    // upload and the last download.
    const int n_chunks_want = 8;
    int cc = ((n_chan + n_chunks_want - 1) / n_chunks_want + 31) / 32 * 32;
    if (cc > n_chan) cc = n_chan;
    const int n_chunks = (n_chan + cc - 1) / cc;
    const size_t plane_bytes = (size_t)p->geom.N * p->geom.N * 8;
    const size_t b_uv = up((size_t)n_vis * 16), b_fr = up((size_t)n_chan * 8);
    const size_t b_vis = up((size_t)n_vis * cc * 32), b_w = weights ? up((size_t)n_vis * cc * 4) : 0;
    const size_t b_grid = (size_t)n_chan * 4 * plane_bytes;
    const int n_in = n_chunks > 1 ? 2 : 1;                                   // input chunk buffers (double-buffered)
    const size_t total = b_uv + b_fr + n_in * (b_vis + b_w) + up(b_grid);
    if (total > p->ws.cap_stage) {
        if (p->ws.d_stage) cudaFree(p->ws.d_stage);
        p->ws.d_stage = nullptr;
        p->ws.cap_stage = 0;
        cudaError_t e = cudaMalloc(&p->ws.d_stage, total);
        if (e != cudaSuccess) { cudaGetLastError(); set_error("staging allocation failed"); return MWA_GRID_ERR_NOMEM; }
        p->ws.cap_stage = total;
    }
    if (n_chunks > 1 && !p->copy_stream[0]) {
        for (int k = 0; k < 2; ++k)
            if (!cuda_ok(cudaStreamCreateWithFlags(&p->copy_stream[k], cudaStreamNonBlocking), "cudaStreamCreate")) return MWA_GRID_ERR_CUDA;
    }
    char* base = (char*)p->ws.d_stage;
    double* d_uv = (double*)base;
    double* d_fr = (double*)(base + b_uv);
    char* d_in = base + b_uv + b_fr;
    float* d_grid = (float*)(d_in + n_in * (b_vis + b_w));
    if (n_vis > 0 && !cuda_ok(cudaMemcpyAsync(d_uv, uv_f64, (size_t)n_vis * 16, cudaMemcpyHostToDevice, st), "H2D uv")) return MWA_GRID_ERR_CUDA;
    if (!cuda_ok(cudaMemcpyAsync(d_fr, freqs, (size_t)n_chan * 8, cudaMemcpyHostToDevice, st), "H2D freqs")) return MWA_GRID_ERR_CUDA;
    cudaStream_t s_up = n_chunks > 1 ? p->copy_stream[0] : st, s_down = n_chunks > 1 ? p->copy_stream[1] : st;
    std::vector<cudaEvent_t> ev_up(n_chunks, nullptr), ev_done(n_chunks, nullptr);
    bool ok = true;
    int launches = 0;
    auto fail = [&](int code) { rc = code; ok = false; };
    if (n_chunks > 1) {
        for (int k = 0; k < n_chunks && ok; ++k)
            if (cudaEventCreateWithFlags(&ev_up[k], cudaEventDisableTiming) != cudaSuccess ||
                cudaEventCreateWithFlags(&ev_done[k], cudaEventDisableTiming) != cudaSuccess) { set_error("cudaEventCreate failed"); fail(MWA_GRID_ERR_CUDA); }
    }
    for (int k = 0; k < n_chunks && ok; ++k) {
        const int c0 = k * cc, nc = (c0 + cc <= n_chan) ? cc : n_chan - c0;
        char* in = d_in + (size_t)(k % n_in) * (b_vis + b_w);
        float* d_vis = (float*)in;
        float* d_w = weights ? (float*)(in + b_vis) : nullptr;
        if (n_chunks > 1 && k >= 2 && cudaStreamWaitEvent(s_up, ev_done[k - 2], 0) != cudaSuccess) { set_error("cudaStreamWaitEvent failed"); fail(MWA_GRID_ERR_CUDA); break; }
        if (n_vis > 0) {
            // the channel slice of the [row][chan] host arrays: a strided (2-D) copy into a contiguous chunk
            if (nc == n_chan) {                                             // one chunk: plain contiguous copies
                if (!cuda_ok(cudaMemcpyAsync(d_vis, vis_c64, (size_t)n_vis * n_chan * 32, cudaMemcpyHostToDevice, s_up), "H2D vis")) { fail(MWA_GRID_ERR_CUDA); break; }
                if (weights && !cuda_ok(cudaMemcpyAsync(d_w, weights, (size_t)n_vis * n_chan * 4, cudaMemcpyHostToDevice, s_up), "H2D weights")) { fail(MWA_GRID_ERR_CUDA); break; }
            } else {
                if (!cuda_ok(cudaMemcpy2DAsync(d_vis, (size_t)nc * 32, (const char*)vis_c64 + (size_t)c0 * 32, (size_t)n_chan * 32, (size_t)nc * 32,
                                               (size_t)n_vis, cudaMemcpyHostToDevice, s_up), "H2D vis")) { fail(MWA_GRID_ERR_CUDA); break; }
                if (weights && !cuda_ok(cudaMemcpy2DAsync(d_w, (size_t)nc * 4, (const char*)weights + (size_t)c0 * 4, (size_t)n_chan * 4, (size_t)nc * 4,
                                                          (size_t)n_vis, cudaMemcpyHostToDevice, s_up), "H2D weights")) { fail(MWA_GRID_ERR_CUDA); break; }
            }
        }
        float* g = d_grid + (size_t)c0 * 4 * (plane_bytes / 4);
        if (n_chunks > 1) {
            cudaEventRecord(ev_up[k], s_up);
            cudaStreamWaitEvent(st, ev_up[k], 0);
        }
        const int r = grid_device(p, d_uv, d_fr + c0, d_vis, d_w, n_vis, nc, g, st);
        if (r != MWA_GRID_OK) { fail(r); break; }
        launches += p->last_launches;
        if (n_chunks > 1) {
            cudaEventRecord(ev_done[k], st);
            cudaStreamWaitEvent(s_down, ev_done[k], 0);
        }
        if (!cuda_ok(cudaMemcpyAsync((char*)grid_out + (size_t)c0 * 4 * plane_bytes, g, (size_t)nc * 4 * plane_bytes, cudaMemcpyDeviceToHost, s_down),
                     "D2H grid")) { fail(MWA_GRID_ERR_CUDA); break; }
    }
    // synchronous by contract: everything enqueued above has finished when the call returns (also after a failure)
    bool sync_ok = cuda_ok(cudaStreamSynchronize(st), "stream synchronize");
    if (n_chunks > 1) {
        sync_ok = cuda_ok(cudaStreamSynchronize(s_up), "copy stream synchronize") && sync_ok;
        sync_ok = cuda_ok(cudaStreamSynchronize(s_down), "copy stream synchronize") && sync_ok;
        for (int k = 0; k < n_chunks; ++k) {
            if (ev_up[k]) cudaEventDestroy(ev_up[k]);
            if (ev_done[k]) cudaEventDestroy(ev_done[k]);
        }
    }
    p->last_launches = launches;
    if (!ok) return rc;
    return sync_ok ? MWA_GRID_OK : MWA_GRID_ERR_CUDA;
}

}  // extern "C"
