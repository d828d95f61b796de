// k_chanws.cu - K6, the warp-specialised channel-SIMD gridder (a2 + a4 + a5) for finely channelised data (C4).
//
// Same ownership idea as K5 (k_chan.cu): the 32 lanes of a warp are 32 ADJACENT CHANNELS (768 channels
// of 40 kHz see a baseline at almost the same cell, and every channel owns its grid), a warp owns a 4x2-cell block and
// keeps its 8 cells x 4 pol x (re, im) = 64 fp32 accumulators in registers from the first tap to the single store.
// What changed is everything around the FMA loop.  K5 ran its phases (bucket sweep, fp64 index, staging, FMA,
// write-out) one after the other on all warps of a CTA, separated by CTA-wide barriers, and repeated the sweep and
// index work for each 16x4 strip: 5.8 G warp instructions for C4, 80 % of them overhead, issue slot use 42 %
// (profiles/r01_chan_v8_c4x128.md).  K6 is a producer / consumer pipeline with no CTA-wide barrier in steady state
// (profiles/r02_chanws_c4.md: 4.2 G warp instructions, C4 in 8.05 ms against 11.9 ms):
//
//   chan_index_kernel (pre-pass, once per call): the exact fp64 index (index.cuh) of every (row, channel), packed in
//       32 bits (stamp origin + table row per axis), and per (row, 32-channel group) the bounding box of the stamp
//       origins over the group's channels.  After it nothing on the path touches fp64 per sample.
//   chan_list_kernel (pre-pass): one warp per item = (16 x 8 cell tile, 32-channel group) sweeps the uv buckets
//       (k_bin.cu) under the tile with integer box tests and writes the item's hit list (row, 16-bit block mask) into a
//       pool; chan_order_kernel splits the items into those with hits and the empty ones.
//
//   chanws_kernel, persistent, one CTA of 20 warps per SM:
//     warp 16  "sweeper"  claims items with hits four at a time and streams their hit lists into a shared-memory queue
//                         in batches of 16, reading each list in a fixed scattered order (see load_entries); an item
//                         whose list found no room in the pool is swept here instead;
//     warp 17, 18 "stagers"  one batch each in turn: cp.async (LDGSTS) of the 32 channels x 32 B of visibilities, the
//                         packed indices (raw table offsets; the consumer adds its tile term) and the weights of every hit
//                         straight into one of 6 stages, completion signalled on the stage's mbarrier by
//                         cp.async.mbarrier.arrive.noinc - a stager never waits for its copies;
//     warp 0..15 "consumers" (4 x 4 blocks of 4 x 2 cells): wait on the batch's mbarrier (parked try_wait), run the
//                         FFMA2 loop of K5 over the hits that touch their block, release the batch; at the end of an
//                         item put the accumulators into a 128 B-swizzled stage slot and signal the store warp;
//     warp 19  "store"    one thread: one cp.async.bulk.tensor store per (2 tile rows x 32 channels x 4 pol) box through a
//                         4-D tensor map of grid_out with dimension order (u, channel, v, pol), evict-first in L2;
//                         claims the empty items from their own list and zero-fills them with 16 KB boxes from a zero
//                         buffer, paced by the sweeper's progress, involving no other warp.  With accumulate-into the
//                         boxes go out as tensor-map reduce-adds and the empty items are skipped.
//
// No atomics on grid data, every cell of grid_out is written exactly once (R10), the hit order is a pure function
// of the sorted rows, so the grid is bit-identical from run to run.  Registers: the kernel is compiled for 96 per
// thread (640 threads); with setmaxnreg the consumers raise themselves to 104 (64 accumulators + two operand sets, no
// spills) and the four service warps drop to 64: five warps per SM sub-partition, 4 x 104 + 64 <= 512 (an increase
// that the pool cannot serve blocks for ever - a 21st warp would not fit).
#include <cuda.h>

#include <cstdint>

#include "plan.h"

namespace mwa {

constexpr int k6Consumers = 16;                       // consumer warps
constexpr int k6Threads = (k6Consumers + 4) * 32;     // + sweeper, two stagers, store warp
constexpr int k6TileX = 16, k6TileY = 8;
#ifndef K6_ZERO_LEAD_PCT
#define K6_ZERO_LEAD_PCT 5
#endif
#ifndef K6_BATCH
#define K6_BATCH 16
#endif
#ifndef K6_STAGES
#define K6_STAGES 6
#endif
constexpr int k6Batch = K6_BATCH;                     // hits per batch
constexpr int k6Stages = K6_STAGES;                   // batches in flight: 6 x 16 hits (measured on C4: 8 x 8 9.43 ms, 14 x 8 8.44, 7 x 16 8.37, 6 x 16 8.34, 28 x 4 9.8)
constexpr int k6Stagers = 2;                          // stager warps; batch b is staged by stager b % 2 into stage b % 4
#ifndef K6_BATCH_RING
#define K6_BATCH_RING 32
#endif
#ifndef K6_ITEM_RING
#define K6_ITEM_RING 16
#endif
constexpr int k6BatchRing = K6_BATCH_RING;                       // batch descriptors / queue segments between sweeper and stagers
constexpr int k6ItemRing = K6_ITEM_RING;                        // consumer-item descriptors between sweeper and store warp
constexpr int k6ZeroChunk = 16;                       // zero items per claim of the store warp
constexpr unsigned k6ExitItem = 0xffffffffu;
constexpr int k6Drift = 8;                            // largest spread (cells) of the stamp origins over the 32 channels of a fast hit
constexpr int k6PadU = 15 + k6Drift + 1, k6PadV = 7 + k6Drift + 1;   // zero padding in front of a table row (floats)
constexpr int k6Bias = 2048;                          // > any stamp origin (N <= 2048): keeps both halves of a raw offset word positive
constexpr int k6ZeroFloats = 32;                      // all-zero block behind each table (target of a missing lane)
constexpr int k6WoSlots = 2;                          // write-out stage slots; block row r uses slot r & 1, rows r and r + 2 take turns
constexpr int k6WoBytes = k6WoSlots * 32768;          // write-out stage: slots of [pol 4][v 2][chan 32][128 B]
constexpr int k6StageV = k6Batch * 1024, k6StageGeo = k6Batch * 128, k6StageW = k6Batch * 128;
constexpr int k6StageBytes = k6StageV + k6StageGeo + k6StageW;
constexpr int k6ZeroV = 4;                            // rows of a zero-fill box
constexpr int k6ZeroBytes = k6ZeroV * 4096;           // zero buffer: [v 4][chan 32][128 B]
constexpr unsigned k6FlagEnd = 1u, k6FlagExit = 2u;
constexpr unsigned k6Invalid = 0xffffffffu;           // packed index of a dropped sample
constexpr long long k6SpinLimit = 6000000000LL;       // ~3 s of SM clocks: a wait this long is a bug -> abort, never hang

enum { K6_ERR_NONE = 0, K6_ERR_FULL = 1, K6_ERR_EMPTY = 2, K6_ERR_WOFULL = 3, K6_ERR_WOEMPTY = 4, K6_ERR_BATCH = 5,
       K6_ERR_ITEM = 6, K6_ERR_RING = 7 };

struct K6Params {
    GridGeom g;
    const double4* group;        // [n_groups] s_lo, s_hi, s_ref / s_lo, s_ref / s_hi (scale_kernel)
    const int* bucket_start;     // [nb*nb + 1]
    const int* perm;             // [n_vis] sorted position -> row
    const unsigned* pre;         // [n_vis][n_groups * 32] packed indices, by ROW
    const ushort4* bb;           // [n_groups][n_vis] bounding boxes, by SORTED POSITION
    const int* list_cnt;         // [n_items] hits of every item (chan_list_kernel); -1 = no list: the in-kernel sweeper sweeps it
    const unsigned* list_off;    // [n_items] first entry of the item's hit list in the pool
    const int4* c_desc;          // [n_c] (item, hits or -1, list offset, 0) of the items with hits, in item order (chan_order_kernel)
    const unsigned* z_list;      // [n_z] the items nothing reaches, in item order
    const int* n_cz;             // [2] n_c, n_z
    const int* n_hits;           // [1] hits of all items (swept items count 64)
    int* zcounter;               // work counter of the zero list
    const uint2* lists;          // [pool_cap] pool of hit lists: (row, mask) entries, an item's hits contiguous and in sweep order
    unsigned pool_cap;           // entries in the pool; 0 = no lists at all
    int* counter;                // work counter
    int* stats;                  // [8] error, items, items with hits, batches, max hits of an item
    const int* dispatch;         // device-side design choice (AUTO); null = always run
    int dispatch_want;
    const float* vis;            // [n_vis][n_chan][8]
    const float* weights;        // [n_vis][n_chan] or null
    const float* table;          // [(O+1)][W]
    float* grid;                 // [n_chan][4][N][N][2] (zero-fill of untouched items; everything else goes through the tensor map)
    int accumulate;              // 1: grid += (f3 accumulate-into: reduce-add stores, no zero-fill), 0: grid = (R10)
    int n_vis, n_chan, n_groups, nb;
    int ntx, nty;                // tiles per row / column
    int rlu, rlv, n_tu, n_tv;    // padded row lengths and sizes (floats) of the shifted table copies
    long long n_items;
};

struct K6Ctrl {
    unsigned long long full[k6Stages], empty[k6Stages];     // mbarriers: batch staged / batch consumed
    unsigned long long wo_full[k6WoSlots], wo_empty[4];     // mbarriers: slot staged for the store (by the 4 warps of a block row) / block row r's store has been read
    int st_n[k6Stages];
    unsigned st_flags[k6Stages];
    unsigned st_tile[k6Stages];                             // tile term of the batch's raw table-offset words
    unsigned st_mask[k6Stages][k6Batch];
    int q_row[k6BatchRing * k6Batch];
    unsigned q_mask[k6BatchRing * k6Batch];                 // bits 0..15 block mask, bit 16: slow staging path
    int b_n[k6BatchRing];
    unsigned b_flags[k6BatchRing];
    int b_x0[k6BatchRing], b_y0[k6BatchRing], b_g[k6BatchRing];
    unsigned c_item[k6ItemRing];                            // consumer items in order: tx | ty << 10 | group << 20, k6ExitItem = exit
    volatile int pub_batches, pub_c, done_c;
    volatile int c_hits;                                    // sweeper: hits of all items before the one it is on (the global work measure)
    volatile int done_batches[k6Stagers];
    volatile int abort;
    alignas(16) int z_ids[k6ZeroChunk];                     // store warp: the zero items of its current claim
    int stat_hit_items, stat_max_hits, stat_swept_items;    // sweeper's counters for mwa_grid_plan_last_stats
};

// Optional phase timing (build with MWA_EXTRA_NVCC=-DK6_TIMING): clock64 sums per role in stats64[], read back through
// mwa_grid_plan_last_stats slots 8.. ; compiled out of the product build.
#ifdef K6_TIMING
#define K6_TIC(t) const long long t = clock64()
#define K6_TOC(acc, t) acc += clock64() - (t)
#define K6_ADD(slot, v) do { if (lane == 0 && P.stats) atomicAdd(reinterpret_cast<unsigned long long*>(P.stats + 2044) + (slot), (unsigned long long)(v)); } while (0)
#else
#define K6_TIC(t)
#define K6_TOC(acc, t)
#define K6_ADD(slot, v)
#endif

struct K6Layout { size_t wo, ring, zero, tu, tv, ctrl, total; };

__host__ __device__ inline K6Layout k6_layout(int n_tu, int n_tv) {
    K6Layout L;
    L.wo = 0;
    L.ring = L.wo + k6WoBytes;
    L.zero = L.ring + (size_t)k6Stages * k6StageBytes;
    L.tu = L.zero + k6ZeroBytes;
    L.tv = L.tu + (size_t)(n_tu + k6ZeroFloats) * 4;
    L.ctrl = (L.tv + (size_t)(n_tv + k6ZeroFloats) * 4 + 15) & ~size_t(15);
    L.total = L.ctrl + sizeof(K6Ctrl);                      // the base must be 1024 B aligned (checked in the kernel)
    return L;
}

// ------------------------------------------------------------------------------------------------ PTX helpers
typedef unsigned long long u64;

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_tx(unsigned bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try(unsigned bar, unsigned parity) {
    unsigned ok;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
}
// Bounded wait: returns false when the kernel is being aborted (a wait that exceeded k6SpinLimit raises the abort).
// try_wait with a suspend-time hint: the hardware parks the thread until the phase completes or ~1 us has passed, so a
// waiting warp does not take issue slots from the working warps of its scheduler
__device__ __forceinline__ bool mbar_try_park(unsigned bar, unsigned parity) {
    unsigned ok;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok) : "r"(bar), "r"(parity), "r"(1000u) : "memory");
    return ok != 0;
}
__device__ __forceinline__ bool mbar_wait(unsigned bar, unsigned parity, volatile int* abort_flag, int code) {
    if (mbar_try(bar, parity)) return true;
    const long long t0 = clock64();
    for (int spins = 1; !mbar_try_park(bar, parity); ++spins) {
        if (*abort_flag) return false;
        if ((spins & 255) == 0 && clock64() - t0 > k6SpinLimit) { *abort_flag = code; return false; }
    }
    return true;
}
__device__ __forceinline__ bool spin_until_gt(volatile int* var, int value, volatile int* abort_flag, int code) {
    if (*var > value) return true;
    const long long t0 = clock64();
    while (!(*var > value)) {
        if (*abort_flag) return false;
        if (clock64() - t0 > k6SpinLimit) { *abort_flag = code; return false; }
        __nanosleep(64);
    }
    return true;
}
__device__ __forceinline__ void bulk_load(unsigned dst, const void* src, unsigned bytes, unsigned bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
// The grid is written once and never read again by this kernel: its lines are marked evict-first in L2, so the 25.8 GB
// write stream does not push the visibilities (re-read by the 2 - 3 tiles a stamp reaches) out of the cache.
__device__ __forceinline__ u64 l2_policy_evict_first() {
    u64 p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ u64 l2_policy_evict_last() {
    u64 p;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ void tma_store4(const CUtensorMap* m, unsigned src, int d0, int d1, int d2, int d3, u64 policy) {
#ifdef K6_NO_L2_HINTS
    asm volatile("cp.async.bulk.tensor.4d.global.shared::cta.bulk_group [%0, {%1, %2, %3, %4}], [%5];"
                 ::"l"(m), "r"(d0), "r"(d1), "r"(d2), "r"(d3), "r"(src) : "memory");
#else
    asm volatile("cp.async.bulk.tensor.4d.global.shared::cta.bulk_group.L2::cache_hint [%0, {%1, %2, %3, %4}], [%5], %6;"
                 ::"l"(m), "r"(d0), "r"(d1), "r"(d2), "r"(d3), "r"(src), "l"(policy) : "memory");
#endif
}
// the same box as a reduction: grid += stage (fp32 add in L2), through a tensor map whose elements are floats
__device__ __forceinline__ void tma_reduce_add4(const CUtensorMap* m, unsigned src, int d0, int d1, int d2, int d3) {
    asm volatile("cp.reduce.async.bulk.tensor.4d.global.shared::cta.add.tile.bulk_group [%0, {%1, %2, %3, %4}], [%5];"
                 ::"l"(m), "r"(d0), "r"(d1), "r"(d2), "r"(d3), "r"(src) : "memory");
}
__device__ __forceinline__ void k6_unpack2(u64 v, float& a, float& b) { asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v)); }
__device__ __forceinline__ u64 k6_pack2(float a, float b) {
    u64 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b));
    return r;
}
__device__ __forceinline__ void k6_ffma2(u64& d, u64 a, u64 b) { asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(d) : "l"(a), "l"(b)); }

// ------------------------------------------------------------------------------------------------ pre-pass
// One warp per sorted row r, walking the channel groups g, lane = channel.  With origin = i - h (the first cell of the stamp):
//   bb[g][r]   = (min origin_u, max origin_u | slow << 15, min origin_v, max origin_v) over the valid lanes; a group with
//                no valid lane gets min = 0x7fff, which no tile reaches.
//   pre[row][c], fast (row, group): the lane's table offsets with the tile term left out,
//                lo16 = 4 (ru rlu + su (O1 rlu - 1) + k6PadU + k6Bias - origin_u), su = (k6PadU - origin_u) & 3, hi16 likewise
//                for v; the consumer adds 4 (X0 - k6Bias) | 4 (Y0 - k6Bias) << 16 of its tile (tiles start at multiples of
//                16 x 8, so the alignment shifts su, sv do not depend on the tile).
//   pre[row][c], slow (row, group): origin_u | ru << 11 | origin_v << 16 | rv << 27, or k6Invalid for a dropped sample (R11)
//                or a channel beyond n_chan; the stager converts these with explicit range checks.
// slow = some valid channel's sample is dropped, the origins spread over more than k6Drift cells (the zero padding of
// the table copies covers a tile + stamp + k6Drift, so a fast hit can never index outside it), or the group is ragged.
__global__ void __launch_bounds__(256)
chan_index_kernel(GridGeom g, const double4* __restrict__ row_sorted, const double* __restrict__ scale, int n_vis,
                  int n_chan, int n_groups, int rlu, int rlv, unsigned* __restrict__ pre, ushort4* __restrict__ bb,
                  const int* __restrict__ dispatch, int dispatch_want) {
    if (dispatch != nullptr && *dispatch != dispatch_want) return;
    const int lane = threadIdx.x & 31;
    const int warps = (int)(((long long)gridDim.x * blockDim.x) >> 5);
    const int ncp = n_groups * 32, O1 = g.O + 1;
    const unsigned full = 0xffffffffu;
    // a warp takes a sorted row and walks its channel groups (the row record is loaded once, no task division)
    for (int r = (int)(((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5); r < n_vis; r += warps) {
        const double4 rec = row_sorted[r];
        unsigned* pre_row = pre + (size_t)(int)rec.z * ncp;
        for (int grp = 0; grp < n_groups; ++grp) {
            const int c = grp * 32 + lane;
            const bool cvalid = c < n_chan;
            const double sc = __ldg(scale + (cvalid ? c : n_chan - 1));
            SampleIndex s;
            const bool ok = sample_index(rec.x, rec.y, sc, g, s) && cvalid;
            const int ou = s.iu - g.h, ov = s.iv - g.h;
            const unsigned u_min = __reduce_min_sync(full, ok ? (unsigned)ou : 0x7fffu);
            const unsigned u_max = __reduce_max_sync(full, ok ? (unsigned)ou : 0u);
            const unsigned v_min = __reduce_min_sync(full, ok ? (unsigned)ov : 0x7fffu);
            const unsigned v_max = __reduce_max_sync(full, ok ? (unsigned)ov : 0u);
            const bool slow = __ballot_sync(full, cvalid && !ok) != 0u || u_max > u_min + k6Drift || v_max > v_min + k6Drift ||
                              grp * 32 + 32 > n_chan;                  // a ragged last group is staged lane by lane as well
            unsigned word = k6Invalid;
            if (ok) {
                if (slow) word = (unsigned)ou | ((unsigned)s.ru << 11) | ((unsigned)ov << 16) | ((unsigned)s.rv << 27);
                else {
                    const int su = (k6PadU - ou) & 3, sv = (k6PadV - ov) & 1;
                    const int lo = s.ru * rlu + su * (O1 * rlu - 1) + k6PadU + k6Bias - ou;
                    const int hi = s.rv * rlv + sv * (O1 * rlv - 1) + k6PadV + k6Bias - ov;
                    word = (unsigned)(lo * 4) | ((unsigned)(hi * 4) << 16);
                }
            }
            pre_row[c] = word;
            if (lane == 0)
                bb[(size_t)grp * n_vis + r] = make_ushort4((unsigned short)u_min, (unsigned short)(u_max | (slow ? 0x8000u : 0u)),
                                                            (unsigned short)v_min, (unsigned short)v_max);
        }
    }
}

// ------------------------------------------------------------------------------------------------ the sweep
// Item = (16 x 8 tile at X0, Y0; channel group grp).  Its bucket window at the reference scale is K5's conservative
// back-projection: il, ih = s_ref / s_lo, s_ref / s_hi of the group (NaN = scan every bucket).
struct K6Item { int X0, Y0, grp, wx0, wx1, wy0, wy1; };

__device__ __forceinline__ K6Item k6_describe(const K6Params& P, int X0, int Y0, int grp, double il, double ih) {
    K6Item it;
    it.X0 = X0; it.Y0 = Y0; it.grp = grp;
    it.wx0 = 0; it.wx1 = P.nb - 1; it.wy0 = 0; it.wy1 = P.nb - 1;
    if (il == il && ih == ih) {
        const double halfN = (double)(P.g.N / 2);
        const double pad = (double)P.g.h + 1.25;
        const double ax = (double)X0 - halfN - pad, bxx = (double)(X0 + k6TileX - 1) - halfN + pad;
        const double ay = (double)Y0 - halfN - pad, byy = (double)(Y0 + k6TileY - 1) - halfN + pad;
        const double ib = 1.0 / kBucketCells, top = (double)(P.nb - 1);
        it.wx0 = (int)fmin(fmax(floor((fmin(ax * il, ax * ih) + halfN) * ib), 0.0), top);
        it.wx1 = (int)fmin(fmax(floor((fmax(bxx * il, bxx * ih) + halfN) * ib), 0.0), top);
        it.wy0 = (int)fmin(fmax(floor((fmin(ay * il, ay * ih) + halfN) * ib), 0.0), top);
        it.wy1 = (int)fmin(fmax(floor((fmax(byy * il, byy * ih) + halfN) * ib), 0.0), top);
    }
    return it;
}

// Item numbering: tile column fastest, then the tile row, then the channel group: neighbouring tiles and tile rows are
// worked on at about the same time and share their halo rows in L2 (with the tile row outermost the call was 0.5 ms
// slower).  The items of the LAST group are re-ordered heaviest first by chan_tail_sort_kernel.
__device__ __forceinline__ void k6_item_decode(const K6Params& P, int item, int& tx, int& ty, int& grp) {
    tx = item % P.ntx; ty = (item / P.ntx) % P.nty; grp = item / (P.ntx * P.nty);
#ifndef K6_NO_TX_INTERLEAVE
    // The four items of a claim run one after the other on one SM; horizontally adjacent tiles share halo rows, which L2
    // keeps for tens of microseconds only.  Within a tile row the columns are therefore taken in the order 0, 4, 8, ...,
    // 1, 5, 9, ...: neighbouring tiles go to different SMs at about the same time.
    if ((P.ntx & 3) == 0 && P.ntx >= 16) {
        const int q = P.ntx >> 2;
        tx = (tx % q) * 4 + tx / q;
    }
#endif
}

// One warp walks the sorted rows of the item's bucket window (lane = candidate, 128 candidates' bounding boxes in
// flight), tests them against the tile with integer compares and calls emit(hit, row, mask, ballot, popc(ballot)) for
// every 32 candidates with at least one hit, in sorted-row order.  mask: bits 0..15 = the 4 x 4 blocks (4 x 2 cells)
// the bounding box of the stamps touches, bit 16 = slow staging path.  Returns false as soon as emit does.
template <typename Emit>
__device__ __forceinline__ bool k6_sweep(const K6Params& P, const K6Item& it, int lane, Emit&& emit) {
    const unsigned full = 0xffffffffu;
    const int W = P.g.W, X0 = it.X0, Y0 = it.Y0;
    const ushort4* bbg = P.bb + (size_t)it.grp * P.n_vis;
    for (int rg = it.wy0; rg <= it.wy1; rg += 32) {
        int k0 = 0, len = 0;
        if (rg + lane <= it.wy1) {                                           // lane = bucket row rg + lane
            k0 = __ldg(P.bucket_start + (rg + lane) * P.nb + it.wx0);
            len = __ldg(P.bucket_start + (rg + lane) * P.nb + it.wx1 + 1) - k0;
        }
        int incl = len;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(full, incl, o);
            if (lane >= o) incl += t;
        }
        const int total = __shfl_sync(full, incl, 31);
        const int excl = incl - len;
        for (int cb = 0; cb < total; cb += 128) {
            uint2 bq[4];
            int rowq[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int f = cb + 32 * u + lane;
                int lo = 0;                                                  // smallest bucket row with incl > f
#pragma unroll
                for (int st = 16; st > 0; st >>= 1) {
                    const int t = __shfl_sync(full, incl, lo + st - 1);
                    if (t <= f) lo += st;
                }
                lo = min(lo, 31);
                const int rk0 = __shfl_sync(full, k0, lo), rex = __shfl_sync(full, excl, lo);
                bq[u] = make_uint2(0x00007fffu, 0x00007fffu);                // empty box (min 0x7fff, max 0): reaches no tile
                rowq[u] = 0;
                if (f < total) {
                    const int kpos = rk0 + (f - rex);
                    bq[u] = __ldg(reinterpret_cast<const uint2*>(bbg + kpos));
                    rowq[u] = __ldg(P.perm + kpos);
                }
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                if (cb + 32 * u >= total) break;
                const int u_min = (int)(bq[u].x & 0xffffu), u_max = (int)((bq[u].x >> 16) & 0x7fffu);
                const int v_min = (int)(bq[u].y & 0xffffu), v_max = (int)(bq[u].y >> 16);
                const bool hit = u_min <= X0 + k6TileX - 1 && u_max + W - 1 >= X0 && v_min <= Y0 + k6TileY - 1 && v_max + W - 1 >= Y0;
                unsigned mask = 0u;
                if (hit) {
                    const int bxl = max(0, (u_min - X0) >> 2), bxh = min(3, (u_max + W - 1 - X0) >> 2);
                    const int byl = max(0, (v_min - Y0) >> 1), byh = min(3, (v_max + W - 1 - Y0) >> 1);
                    const unsigned mu = (2u << bxh) - (1u << bxl);
                    const unsigned mv = 0x1111u & ((1u << (4 * (byh + 1))) - (1u << (4 * byl)));
                    mask = mu * mv | ((bq[u].x & 0x80000000u) ? 0x10000u : 0u);
                }
                const unsigned hm = __ballot_sync(full, hit);
                const int n_new = __popc(hm);
                if (n_new == 0) continue;
                if (!emit(hit, rowq[u], mask, hm, n_new)) return false;
            }
        }
    }
    return true;
}

// Second pre-pass: one warp per item sweeps it and writes its hit list (row, mask) into a pool.  The slot of an item is
// reserved with one atomicAdd of an upper bound that costs nothing to compute - the number of sorted rows in the item's
// bucket window (every hit is one of them) - so lists of any length are contiguous and written in one sweep; where a
// list lands in the pool may differ from run to run, what it holds does not.  An item the pool has no room for gets the
// count -1 and is swept by chanws_kernel's own sweeper instead.  Runs with thousands of warps in flight, which hides the
// L2 round trips a single in-kernel sweeper warp pays one after the other (4.6 us per item measured).
__global__ void __launch_bounds__(256)
chan_list_kernel(const __grid_constant__ K6Params P, int* __restrict__ list_cnt, unsigned* __restrict__ list_off,
                 uint2* __restrict__ pool, unsigned long long* __restrict__ cursor) {
    if (P.dispatch != nullptr && *P.dispatch != P.dispatch_want) return;
    const unsigned full = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    const int warps = (gridDim.x * blockDim.x) >> 5;
    const int n_items = (int)P.n_items;
    const unsigned lt_mask = (1u << lane) - 1u;
    for (int item = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; item < n_items; item += warps) {
        int tx, ty, grp;
        k6_item_decode(P, item, tx, ty, grp);
        const double4 gi = P.group[grp];
        const K6Item it = k6_describe(P, tx * k6TileX, ty * k6TileY, grp, gi.z, gi.w);
        int cand = 0;
        for (int rg = it.wy0 + lane; rg <= it.wy1; rg += 32)
            cand += __ldg(P.bucket_start + rg * P.nb + it.wx1 + 1) - __ldg(P.bucket_start + rg * P.nb + it.wx0);
        cand = __reduce_add_sync(full, cand);
        if (cand == 0) {
            if (lane == 0) { list_cnt[item] = 0; list_off[item] = 0u; }
            continue;
        }
        unsigned long long base = 0ull;
        if (lane == 0) base = atomicAdd(cursor, (unsigned long long)cand);
        base = __shfl_sync(full, base, 0);
        if (base + (unsigned long long)cand > (unsigned long long)P.pool_cap) {
            if (lane == 0) { list_cnt[item] = -1; list_off[item] = 0u; }
            continue;
        }
        uint2* dst = pool + base;
        int cnt = 0;
        k6_sweep(P, it, lane, [&](bool hit, int row, unsigned mask, unsigned hm, int n_new) -> bool {
            if (hit) dst[cnt + __popc(hm & lt_mask)] = make_uint2((unsigned)row, mask);
            cnt += n_new;
            return true;
        });
        if (lane == 0) { list_cnt[item] = cnt; list_off[item] = (unsigned)base; }
    }
}

// Third pre-pass: splits the items into those with hits (c_desc: item, hit count, list offset - what the sweeper of
// chanws_kernel claims, four at a time) and those nothing reaches (z_list - what its store warp claims), both in item
// order, so neighbouring tiles are still worked on at about the same time and share their halo rows in L2.
// A block takes `per_block` consecutive items, publishes its number of items with hits in blk_state (zeroed by the
// call's memset; flag bit 30) and sums the counts of the blocks before it (they were scheduled before it, so the wait
// cannot deadlock) - a one-level decoupled scan, enough for the <= 1024 blocks the launcher uses.  The same scan runs over the hit counts: c_desc.w is the
// number of hits of all items before this one, the work measure that paces the zero-fill.
constexpr int k6OrderBlocksMax = 1024;                 // two state arrays of this length in d_misc (counts, hits)
constexpr int k6OrderFlag = 1 << 30;

__global__ void __launch_bounds__(1024)
chan_order_kernel(const int* __restrict__ list_cnt, const unsigned* __restrict__ list_off, int n_items, int per_block,
                  int4* __restrict__ c_desc, unsigned* __restrict__ z_list, int* __restrict__ n_cz, int* __restrict__ n_hits,
                  int first_item_of_last_group, int* __restrict__ tail_start, volatile int* blk_state,
                  const int* __restrict__ dispatch, int dispatch_want) {
    if (dispatch != nullptr && *dispatch != dispatch_want) return;
    __shared__ int s_warp[32], s_hwarp[32];
    __shared__ int s_prefix, s_hprefix;
    const unsigned full = 0xffffffffu;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int b = blockIdx.x;
    const int i0 = min(n_items, b * per_block), i1 = min(n_items, i0 + per_block);
    volatile int* hit_state = blk_state + k6OrderBlocksMax;          // second scan: the hits of the items (the work measure)
    // a swept item (-1: its list is unknown) counts as 64 hits in the work measure
    int nz = 0, nh = 0;
    for (int i = i0 + tid; i < i1; i += 1024) {
        const int c = list_cnt[i];
        nz += c != 0 ? 1 : 0;
        nh += c < 0 ? 64 : c;
    }
    nz = __reduce_add_sync(full, nz);
    nh = __reduce_add_sync(full, nh);
    if (lane == 0) { s_warp[warp] = nz; s_hwarp[warp] = nh; }
    __syncthreads();
    if (warp == 0) {
        const int total = __reduce_add_sync(full, s_warp[lane]), htotal = __reduce_add_sync(full, s_hwarp[lane]);
        if (lane == 0) { blk_state[b] = total | k6OrderFlag; hit_state[b] = htotal | k6OrderFlag; }
        int sum = 0, hsum = 0;
        for (int j0 = 0; j0 < b; j0 += 32) {
            const int j = j0 + lane;
            int v = 0, h = 0;
            if (j < b) {
                do { v = blk_state[j]; } while (!(v & k6OrderFlag));
                do { h = hit_state[j]; } while (!(h & k6OrderFlag));
                v &= ~k6OrderFlag; h &= ~k6OrderFlag;
            }
            sum += v; hsum += h;
        }
        sum = __reduce_add_sync(full, sum);
        hsum = __reduce_add_sync(full, hsum);
        if (lane == 0) {
            s_prefix = sum; s_hprefix = hsum;
            if (b == (int)gridDim.x - 1) { n_cz[0] = sum + total; n_cz[1] = n_items - (sum + total); *n_hits = hsum + htotal; }
        }
    }
    __syncthreads();
    int cb = s_prefix, hb = s_hprefix;                               // items with hits / hits before the current chunk
    const unsigned lt_mask = (1u << lane) - 1u;
    for (int s0 = i0; s0 < i1; s0 += 1024) {
        const int i = s0 + tid;
        const bool valid = i < i1;
        const int cnt = valid ? list_cnt[i] : 0;
        const int hits = cnt < 0 ? 64 : cnt;
        const unsigned bm = __ballot_sync(full, valid && cnt != 0);
        int hincl = hits;                                            // inclusive scan of the hits inside the warp
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int u = __shfl_up_sync(full, hincl, o);
            if (lane >= o) hincl += u;
        }
        __syncthreads();                                             // s_warp / s_hwarp are free again
        if (lane == 0) s_warp[warp] = __popc(bm);
        if (lane == 31) s_hwarp[warp] = hincl;
        __syncthreads();
        const int t = s_warp[lane], ht = s_hwarp[lane];
        int incl = t, hinc2 = ht;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int u = __shfl_up_sync(full, incl, o), hu = __shfl_up_sync(full, hinc2, o);
            if (lane >= o) { incl += u; hinc2 += hu; }
        }
        const int before = __shfl_sync(full, incl - t, warp);        // items with hits in the warps before this one
        const int hbefore = __shfl_sync(full, hinc2 - ht, warp);     // their hits
        const int chunk_total = __shfl_sync(full, incl, 31), hchunk_total = __shfl_sync(full, hinc2, 31);
        if (valid) {
            const int cpos = cb + before + __popc(bm & lt_mask);     // items with hits before item i
            if (i == first_item_of_last_group) *tail_start = cpos;   // where the last channel group begins in c_desc
            if (cnt != 0) c_desc[cpos] = make_int4(i, cnt, (int)list_off[i], hb + hbefore + hincl - hits);   // .w: hits before it
            else z_list[i - cpos] = (unsigned)i;
        }
        cb += chunk_total;
        hb += hchunk_total;
    }
}

// Fourth pre-pass, one block: the items with hits of the LAST channel group - the tail of c_desc, which is in item order -
// are sorted heaviest first (by weight class).  The dense centre tiles of a group take 0.1 - 0.2 ms
// each and are claimed four at a time; in item order the last group's centre rows come 0.15 ms before the end of the
// kernel and the SMs that claimed them finished 0.3 - 0.4 ms after all others (measured with per-CTA end times).  Heaviest
// first, every SM starts the last group with dense items and the sparse ones fill the end evenly.
constexpr int k6TailMax = 8192;                                      // entries sorted (128 KB of entries + 64 KB of keys in shared memory)

__global__ void __launch_bounds__(1024)
chan_tail_sort_kernel(int4* __restrict__ c_desc, const int* __restrict__ n_cz, const int* __restrict__ tail_start,
                      const int* __restrict__ dispatch, int dispatch_want) {
    if (dispatch != nullptr && *dispatch != dispatch_want) return;
    extern __shared__ __align__(16) unsigned char s_raw[];
    int4* s_e = reinterpret_cast<int4*>(s_raw);                                   // the entries, in item order
    unsigned long long* s_k = reinterpret_cast<unsigned long long*>(s_raw + (size_t)k6TailMax * 16);   // sort keys
    const int n_c = n_cz[0];
    const int lo = max(*tail_start, n_c - k6TailMax), n = n_c - lo;
    if (n < 2) return;
    // a counting sort by weight class (floor(log2 hits), heaviest class first; swept items, -1, in the lightest): within a
    // factor of two of heaviest-first, which is all the balancing needs, and three passes instead of a 78-step network.
    // The order inside a class is whatever the atomics give - the order of the ITEMS does not touch any grid value.
    __shared__ int s_hist[32], s_cur[32];
    if (threadIdx.x < 32) s_hist[threadIdx.x] = 0;
    __syncthreads();
    for (int i = threadIdx.x; i < n; i += 1024) {
        const int4 e = c_desc[lo + i];
        s_e[i] = e;
        atomicAdd(&s_hist[31 - __clz(max(e.y, 1))], 1);
    }
    __syncthreads();
    if (threadIdx.x < 32) {
        int start = 0;
        for (int c = 31; c > (int)threadIdx.x; --c) start += s_hist[c];
        s_cur[threadIdx.x] = start;
    }
    __syncthreads();
    for (int i = threadIdx.x; i < n; i += 1024) s_k[atomicAdd(&s_cur[31 - __clz(max(s_e[i].y, 1))], 1)] = (unsigned long long)i;
    __syncthreads();
    // written back interleaved: the sweepers claim four consecutive entries at a time, so claim k gets the entries k,
    // k + n/4, k + n/2, k + 3n/4 of the sorted order - one of the heaviest with three lighter ones, not the four heaviest
    const int n4 = n & ~3, q = n4 >> 2;
    for (int i = threadIdx.x; i < n; i += 1024) {
        const int src = i < n4 ? (i & 3) * q + (i >> 2) : i;
        c_desc[lo + i] = s_e[(int)(s_k[src] & 0xffffffffu)];
    }
}

// ------------------------------------------------------------------------------------------------ main kernel
template <bool HAS_W>
__global__ void __launch_bounds__(k6Threads, 1)
chanws_kernel(const __grid_constant__ K6Params P, const __grid_constant__ CUtensorMap map_out,
              const __grid_constant__ CUtensorMap map_zero, const __grid_constant__ CUtensorMap map_acc) {
    if (P.dispatch != nullptr && *P.dispatch != P.dispatch_want) return;
    extern __shared__ __align__(1024) unsigned char smem_dyn[];
    unsigned char* base = smem_dyn;
    if ((smem_u32(base) & 1023u) != 0u) {                             // the swizzled TMA stage needs it; never seen, never silent
        if (threadIdx.x == 0 && P.stats) atomicMax(P.stats, 100);
        return;
    }
    const K6Layout L = k6_layout(P.n_tu, P.n_tv);
    float* tu = reinterpret_cast<float*>(base + L.tu);
    float* tv = reinterpret_cast<float*>(base + L.tv);
    K6Ctrl& S = *reinterpret_cast<K6Ctrl*>(base + L.ctrl);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int W = P.g.W, O1 = P.g.O + 1, N = P.g.N;
    const unsigned full = 0xffffffffu;

    // ---- set-up by all 20 warps: shifted zero-padded table copies (as K5), zero buffer, control block, mbarriers
    //   tu[s][r][q] = Tp_u[r][q + s], Tp_u[r][k6PadU + t] = T[r][t]   s = 0..3 (LDS.128 alignment)
    //   tv[s][r][q] = Tp_v[r][q + s], Tp_v[r][k6PadV + t] = T[r][t]   s = 0..1 (LDS.64 alignment)
    for (int k = tid; k < P.n_tu + k6ZeroFloats; k += k6Threads) {
        float v = 0.0f;
        if (k < P.n_tu) {
            const int q = k % P.rlu, r = (k / P.rlu) % O1, s = k / (P.rlu * O1);
            const int t = q + s - k6PadU;
            if (t >= 0 && t < W) v = P.table[r * W + t];
        }
        tu[k] = v;
    }
    for (int k = tid; k < P.n_tv + k6ZeroFloats; k += k6Threads) {
        float v = 0.0f;
        if (k < P.n_tv) {
            const int q = k % P.rlv, r = (k / P.rlv) % O1, s = k / (P.rlv * O1);
            const int t = q + s - k6PadV;
            if (t >= 0 && t < W) v = P.table[r * W + t];
        }
        tv[k] = v;
    }
    for (int k = tid; k < k6ZeroBytes / 4; k += k6Threads) reinterpret_cast<float*>(base + L.zero)[k] = 0.0f;
    for (int k = tid; k < (int)(sizeof(K6Ctrl) / 4); k += k6Threads) reinterpret_cast<int*>(&S)[k] = 0;
    __syncthreads();
    if (tid == 0) {
        for (int s = 0; s < k6Stages; ++s) {
            mbar_init(smem_u32(&S.full[s]), 33); mbar_init(smem_u32(&S.empty[s]), k6Consumers);   // 32 cp.async arrivals + 1
        }
        for (int r = 0; r < k6WoSlots; ++r) mbar_init(smem_u32(&S.wo_full[r]), 4);
        for (int r = 0; r < 4; ++r) mbar_init(smem_u32(&S.wo_empty[r]), 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");      // zero buffer and barriers visible to the async proxy
    __syncthreads();

    volatile int* abort_flag = &S.abort;
    const unsigned ring_s = smem_u32(base + L.ring);

    if (warp < k6Consumers) {
        // =========================================================================================== consumers
        asm volatile("setmaxnreg.inc.sync.aligned.u32 104;");
        const int bx = warp & 3, by = warp >> 2;
        const unsigned wbit = (unsigned)warp;                           // bit by * 4 + bx of a hit mask
        const unsigned tu_s = smem_u32(tu) + 16u * bx, tv_s = smem_u32(tv) + 8u * by;
        // the lane's two 16 B chunks of a 128 B stage row: chunk (2 bx + k) ^ (row & 7), row & 7 = lane & 7
        const unsigned wo_s = smem_u32(base + L.wo) + 32768u * (by & 1) + 128u * lane;
        const unsigned wo_c0 = wo_s + 16u * ((2u * bx) ^ (lane & 7u)), wo_c1 = wo_s + 16u * ((2u * bx + 1u) ^ (lane & 7u));
        u64 acc[2][4][4];                                               // [row i][col j][pol] = (re, im) of the lane's channel
#pragma unroll
        for (int i = 0; i < 2; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j)
#pragma unroll
                for (int p = 0; p < 4; ++p) acc[i][j][p] = 0ull;
        int n_written = 0;
        long long t_full = 0, t_visit = 0, t_woe = 0, t_wo = 0, n_vis_cnt = 0, n_bat = 0;
        (void)t_full; (void)t_visit; (void)t_woe; (void)t_wo; (void)n_vis_cnt; (void)n_bat;
        for (int k = 0;; ++k) {
            const int s = k % k6Stages;
            K6_TIC(c0);
            if (!mbar_wait(smem_u32(&S.full[s]), (unsigned)((k / k6Stages) & 1), abort_flag, K6_ERR_FULL)) break;
            K6_TOC(t_full, c0);
            K6_TIC(c1);
            const unsigned flags = S.st_flags[s];
            if (flags & k6FlagExit) break;
            unsigned m = __ballot_sync(full, lane < k6Batch && ((S.st_mask[s][lane] >> wbit) & 1u));
            const unsigned tc = S.st_tile[s];                           // 4 (X0 - k6Bias) | 4 (Y0 - k6Bias) << 16: completes a raw offset word
            const unsigned zs_s = ring_s + (unsigned)s * k6StageBytes + 16u * lane;   // [hit][half][lane][16 B]: conflict-free LDS.128
            const unsigned geo_s = ring_s + (unsigned)s * k6StageBytes + k6StageV + 4u * lane;
            const unsigned wt_s = geo_s + k6StageGeo;
#ifdef K6_ABLATE_FMA
            m = 0u;
#endif
            if (m != 0u) {
                // software pipeline over the set bits of m, two visits per trip with two register sets (as K5 phase B)
#define K6_NEXT(mm, prev) ((mm) ? (int)(__ffs(mm) - 1) : (prev)); (mm) &= (mm) - 1u
#define K6_LOAD(h, g, Z0, Z1, Z2, Z3, U0, U1, U2, U3, V0, V1, WT)                                                         \
    asm volatile("ld.shared.v2.b64 {%0, %1}, [%2];" : "=l"(Z0), "=l"(Z1) : "r"(zs_s + 1024u * (h)));                       \
    asm volatile("ld.shared.v2.b64 {%0, %1}, [%2];" : "=l"(Z2), "=l"(Z3) : "r"(zs_s + 1024u * (h) + 512u));                \
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(U0), "=f"(U1), "=f"(U2), "=f"(U3) : "r"(tu_s + ((g) & 0xffffu))); \
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(V0), "=f"(V1) : "r"(tv_s + ((g) >> 16)));                       \
    if (HAS_W) asm volatile("ld.shared.f32 %0, [%1];" : "=f"(WT) : "r"(wt_s + 128u * (h)));
#define K6_FMA(Z0, Z1, Z2, Z3, U0, U1, U2, U3, V0, V1, WT)                                                                \
    {                                                                                                                     \
        const float kvw[2] = {HAS_W ? V0 * WT : V0, HAS_W ? V1 * WT : V1};                                                \
        const float kuu[4] = {U0, U1, U2, U3};                                                                            \
        _Pragma("unroll") for (int i = 0; i < 2; ++i) _Pragma("unroll") for (int j = 0; j < 4; ++j) {                      \
            const float kq = kvw[i] * kuu[j];                                                                             \
            const u64 kk = k6_pack2(kq, kq);                                                                              \
            k6_ffma2(acc[i][j][0], kk, Z0);                                                                               \
            k6_ffma2(acc[i][j][1], kk, Z1);                                                                               \
            k6_ffma2(acc[i][j][2], kk, Z2);                                                                               \
            k6_ffma2(acc[i][j][3], kk, Z3);                                                                               \
        }                                                                                                                 \
    }
                const int cnt = __popc(m);
#ifdef K6_TIMING
                n_vis_cnt += cnt;
#endif
                u64 az0, az1, az2, az3, bz0, bz1, bz2, bz3;
                float au0, au1, au2, au3, av0, av1, aw = 1.0f, bu0, bu1, bu2, bu3, bv0, bv1, bw = 1.0f;
                const int h0 = K6_NEXT(m, 0);
                int h1 = K6_NEXT(m, h0);
                int h2 = K6_NEXT(m, h1);
                unsigned g1, g2;
                {
                    unsigned g0;
                    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(g0) : "r"(geo_s + 128u * h0));
                    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(g1) : "r"(geo_s + 128u * h1));
                    g0 += tc; g1 += tc;
                    K6_LOAD(h0, g0, az0, az1, az2, az3, au0, au1, au2, au3, av0, av1, aw)
                }
#pragma unroll 1
                for (int v = 0; v < cnt; v += 2) {
                    K6_LOAD(h1, g1, bz0, bz1, bz2, bz3, bu0, bu1, bu2, bu3, bv0, bv1, bw)
                    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(g2) : "r"(geo_s + 128u * h2));
                    g2 += tc;
                    const int h3 = K6_NEXT(m, h2);
                    K6_FMA(az0, az1, az2, az3, au0, au1, au2, au3, av0, av1, aw)
                    if (v + 1 >= cnt) break;
                    K6_LOAD(h2, g2, az0, az1, az2, az3, au0, au1, au2, au3, av0, av1, aw)
                    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(g1) : "r"(geo_s + 128u * h3));
                    g1 += tc;
                    const int h4 = K6_NEXT(m, h3);
                    K6_FMA(bz0, bz1, bz2, bz3, bu0, bu1, bu2, bu3, bv0, bv1, bw)
                    h1 = h3;
                    h2 = h4;
                }
#undef K6_NEXT
#undef K6_LOAD
#undef K6_FMA
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(smem_u32(&S.empty[s]));          // this warp has read everything it needs of the batch
            K6_TOC(t_visit, c1);
#ifdef K6_TIMING
            ++n_bat;
#endif
            if (flags & k6FlagEnd) {
                // ---- a5: accumulators -> swizzled stage of this block row; the store warp issues the TMA store
                K6_TIC(c2);
                // block rows by and by ^ 2 take turns on slot by & 1 (0, 2, 0, 2, ... item after item): the slot is free when
                // the store of the OTHER row's last use has been read - rows 2, 3 wait for rows 0, 1 of this item, rows 0, 1 for
                // rows 2, 3 of the item before (the store warp keeps that order, so the own last use has been read as well)
                if (!mbar_wait(smem_u32(&S.wo_empty[by ^ 2]), (unsigned)((n_written & 1) ^ (by < 2 ? 1 : 0)), abort_flag, K6_ERR_WOEMPTY)) break;
                K6_TOC(t_woe, c2);
                K6_TIC(c3);
#pragma unroll
                for (int pol = 0; pol < 4; ++pol)
#pragma unroll
                    for (int i = 0; i < 2; ++i) {
                        float a0, a1, a2, a3, b0, b1, b2, b3;
                        k6_unpack2(acc[i][0][pol], a0, a1); k6_unpack2(acc[i][1][pol], a2, a3);
                        k6_unpack2(acc[i][2][pol], b0, b1); k6_unpack2(acc[i][3][pol], b2, b3);
                        const unsigned ro = (unsigned)(pol * 2 + i) * 4096u;
                        asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(wo_c0 + ro), "f"(a0), "f"(a1), "f"(a2), "f"(a3) : "memory");
                        asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(wo_c1 + ro), "f"(b0), "f"(b1), "f"(b2), "f"(b3) : "memory");
                        acc[i][0][pol] = 0ull; acc[i][1][pol] = 0ull; acc[i][2][pol] = 0ull; acc[i][3][pol] = 0ull;
                    }
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                __syncwarp();
                if (lane == 0) mbar_arrive(smem_u32(&S.wo_full[by & 1]));
                ++n_written;
                K6_TOC(t_wo, c3);
            }
        }
        K6_ADD(0, t_full); K6_ADD(1, t_visit); K6_ADD(2, t_woe); K6_ADD(3, t_wo); K6_ADD(4, n_vis_cnt); K6_ADD(5, n_bat);
    } else {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 64;");
        const int role = warp - k6Consumers;
        if (role == 0) {
            // =========================================================================================== sweeper
            // Streams the per-item hit lists of chan_list_kernel into the queue: nothing here waits on global memory,
            // because items are claimed four at a time with the next claim, its hit counts and the next item's list
            // entries already in flight.  An item whose list overflowed its slot (dense tiles) is swept here instead.
            int b_next = 0;              // global index of the first batch of the current item
            int n_pub = 0;               // batches published so far (= b_next + complete batches of the current item)
            int i_pub = 0;               // items published so far
            bool alive = true;
            long long t_sw_ring = 0, t_sw_item = 0, t_sw_all = 0, t_sw_atomic = 0, t_sw_desc = 0, t_sw_loop = 0;
            (void)t_sw_ring; (void)t_sw_item; (void)t_sw_all; (void)t_sw_atomic; (void)t_sw_desc; (void)t_sw_loop;
            K6_TIC(sw0);
            // wait until batch b's queue segment and descriptor may be reused (batch b - ring has been staged)
            auto batch_slot_free = [&](int b) -> bool {
                const int old = b - k6BatchRing;
                if (old < 0) return true;
                K6_TIC(r0);
                const bool okr = spin_until_gt(&S.done_batches[old % k6Stagers], old / k6Stagers, abort_flag, K6_ERR_RING);
                K6_TOC(t_sw_ring, r0);
                return okr;
            };
            auto publish_batches = [&](int upto, int n_last, unsigned flags_last, int x0, int y0, int grp) {
                // publishes batches [n_pub, upto]; all but the last are full and carry no flag
                if (lane == 0) {
                    for (int b = n_pub; b <= upto; ++b) {
                        const int q = b % k6BatchRing;
                        S.b_n[q] = b == upto ? n_last : k6Batch;
                        S.b_flags[q] = b == upto ? flags_last : 0u;
                        S.b_x0[q] = x0; S.b_y0[q] = y0; S.b_g[q] = grp;
                    }
                }
                __syncwarp();
                __threadfence_block();
                if (lane == 0) S.pub_batches = upto + 1;
                n_pub = upto + 1;
            };
            // consumer item (in order), or with exit = true the exit marker behind the last one
            auto publish_item = [&](int x0, int y0, int grp, bool exit) -> bool {
                const unsigned word = exit ? k6ExitItem : ((unsigned)(x0 / k6TileX) | ((unsigned)(y0 / k6TileY) << 10) | ((unsigned)grp << 20));
                K6_TIC(r1);
                if (!spin_until_gt(&S.done_c, i_pub - k6ItemRing, abort_flag, K6_ERR_ITEM)) return false;
                K6_TOC(t_sw_item, r1);
                if (lane == 0) {
                    S.c_item[i_pub % k6ItemRing] = word;
                    __threadfence_block();
                    S.pub_c = i_pub + 1;
                }
                ++i_pub;
                __syncwarp();
                return true;
            };
            const int n_c = __ldg(P.n_cz);
            auto claim = [&]() -> int { return lane == 0 ? atomicAdd(P.counter, 4) : 0; };      // raw: valid in lane 0 only
            // lane k < 4: (item, hit count, list offset) of entry base + k of the list of items with hits
            auto load_desc = [&](int base) -> int4 {
                int4 d = make_int4(0, 0, 0, 0);
                if (lane < 4 && base + lane < n_c && base >= 0) d = __ldg(P.c_desc + base + lane);
                return d;
            };
            // The list is in sorted-row order, i.e. bucket after bucket: consecutive hits fall on the same few 4 x 2 blocks and
            // would keep a few consumer warps busy while the others wait.  It is therefore read in a fixed scattered order,
            // position p -> entry (p * S) mod c with S ~ 0.618 c coprime to c (a low-discrepancy stride: any run of positions
            // is spread over the whole list, hence over the whole tile).  A pure function of the list: still deterministic.
            auto stride_of = [&](int c) -> int {
                if (c < 16) return 1;
                int S = (int)(((long long)c * 618) / 1000) | 1;
                for (;; S += 2) {
                    int a = c, b = S;
                    while (b) { const int t = a % b; a = b; b = t; }
                    if (a == 1) return S;
                }
            };
            auto load_entries = [&](unsigned off, int c, int S, int first, uint2& ea, uint2& eb) {   // list positions first + lane, first + lane + 32
                ea = make_uint2(0u, 0u); eb = ea;
                if (c > 0) {
                    const uint2* src = P.lists + off;
                    const int pa = first + lane, pb = first + lane + 32;
                    if (pa < c) ea = __ldg(src + (int)(((long long)pa * S) % c));
                    if (pb < c) eb = __ldg(src + (int)(((long long)pb * S) % c));
                }
            };
            K6_TIC(r2);
            int ci = __shfl_sync(full, claim(), 0);          // index into c_desc
            K6_TOC(t_sw_atomic, r2);
            int4 d4 = load_desc(ci), d4_n = make_int4(0, 0, 0, 0);
            int base_n = 0;
            int raw_next = claim();
            int sub = 0;
            uint2 ea, eb;
            int S_cur = stride_of(__shfl_sync(full, d4.y, 0));
            load_entries((unsigned)__shfl_sync(full, d4.z, 0), __shfl_sync(full, d4.y, 0), S_cur, 0, ea, eb);
            while (alive && ci < n_c && ci >= 0) {
                // ---- look ahead: the next claim's descriptors (one item after the claim was issued), the next item's entries
                if (sub == 1) {
                    K6_TIC(r3);
                    base_n = __shfl_sync(full, raw_next, 0);
                    K6_TOC(t_sw_atomic, r3);
                    d4_n = load_desc(base_n);
                }
                const int item = __shfl_sync(full, d4.x, sub), c = __shfl_sync(full, d4.y, sub);
                const int hits_before = __shfl_sync(full, d4.w, sub);
                if (lane == 0) S.c_hits = hits_before;
                const unsigned off = (unsigned)__shfl_sync(full, d4.z, sub);
                const int ci_n = sub == 3 ? base_n : ci + 1;
                const bool valid_n = ci_n < n_c && ci_n >= 0;
                const int c_n = valid_n ? (sub == 3 ? __shfl_sync(full, d4_n.y, 0) : __shfl_sync(full, d4.y, (sub + 1) & 3)) : 0;
                const unsigned off_n = (unsigned)(sub == 3 ? __shfl_sync(full, d4_n.z, 0) : __shfl_sync(full, d4.z, (sub + 1) & 3));
                uint2 ea_n, eb_n;
                const int S_n = stride_of(c_n);
                load_entries(off_n, c_n, S_n, 0, ea_n, eb_n);
                // ---- this item
                int tx, ty, grp;
        k6_item_decode(P, item, tx, ty, grp);
                const int X0 = tx * k6TileX, Y0 = ty * k6TileY;
                int cnt = 0;
                if (c > 0) {
                    // list path: the list is streamed in chunks of 64 hits = 8 batches, the next chunk in flight while this
                    // one goes into the queue.  Per chunk: open the batches (the two youngest cover both stagers), write the
                    // queue and the descriptors lane-parallel, publish everything with one fence
                    K6_TIC(d0);
                    for (int done = 0;;) {
                        const int n_chunk = min(64, c - done);
                        const bool more = done + 64 < c;
                        uint2 fa = make_uint2(0u, 0u), fb = fa;
                        if (more) load_entries(off, c, S_cur, done + 64, fa, fb);
                        const int nbat = (n_chunk + k6Batch - 1) / k6Batch;
                        alive = batch_slot_free(b_next + nbat - 1) && (nbat < 2 || batch_slot_free(b_next + nbat - 2));
                        if (!alive) break;
                        if (lane < n_chunk) {
                            const int slot = ((b_next + lane / k6Batch) % k6BatchRing) * k6Batch + (lane % k6Batch);
                            S.q_row[slot] = (int)ea.x; S.q_mask[slot] = ea.y;
                        }
                        if (lane + 32 < n_chunk) {
                            const int i = lane + 32;
                            const int slot = ((b_next + i / k6Batch) % k6BatchRing) * k6Batch + (i % k6Batch);
                            S.q_row[slot] = (int)eb.x; S.q_mask[slot] = eb.y;
                        }
                        if (lane < nbat) {
                            const int q = (b_next + lane) % k6BatchRing;
                            const bool lastb = lane == nbat - 1;
                            S.b_n[q] = lastb ? n_chunk - (nbat - 1) * k6Batch : k6Batch;
                            S.b_flags[q] = (lastb && !more) ? k6FlagEnd : 0u;
                            S.b_x0[q] = X0; S.b_y0[q] = Y0; S.b_g[q] = grp;
                        }
                        __syncwarp();
                        __threadfence_block();
                        if (lane == 0) S.pub_batches = b_next + nbat;
                        b_next += nbat;
                        n_pub = b_next;
                        if (!more) break;
                        done += 64;
                        ea = fa; eb = fb;
                    }
                    K6_TOC(t_sw_desc, d0);
                    if (!alive) break;
                    if (lane == 0) { S.stat_hit_items += 1; S.stat_max_hits = max(S.stat_max_hits, c); }
                } else {
                    // fallback: the in-kernel sweep (the pool had no room for this item's list)
                    K6_TIC(d1);
                    const double4 gi = P.group[grp];
                    const K6Item it = k6_describe(P, X0, Y0, grp, gi.z, gi.w);
                    int opened = 0;
                    const unsigned lt_mask = (1u << lane) - 1u;
                    alive = k6_sweep(P, it, lane, [&](bool hit, int row, unsigned mask, unsigned hm, int n_new) -> bool {
                        const int need = (cnt + n_new - 1) / k6Batch + 1;    // batches of this item that must be open
                        while (opened < need) {
                            if (!batch_slot_free(b_next + opened)) return false;
                            ++opened;
                        }
                        if (hit) {
                            const int i = cnt + __popc(hm & lt_mask);
                            const int slot = ((b_next + i / k6Batch) % k6BatchRing) * k6Batch + (i % k6Batch);
                            S.q_row[slot] = row;
                            S.q_mask[slot] = mask;
                        }
                        cnt += n_new;
                        const int complete = b_next + (cnt - 1) / k6Batch - 1;    // last batch known to have a successor
                        if (complete >= n_pub) publish_batches(complete, k6Batch, 0u, X0, Y0, grp);
                        return true;
                    });
                    K6_TOC(t_sw_loop, d1);
                    if (!alive) break;
                    // the last batch carries the end flag; an item the sweep found nothing for gets one empty batch, so the
                    // consumers write its zeros through the ordinary path
                    if (cnt == 0 && !batch_slot_free(b_next)) { alive = false; break; }
                    const int last = cnt > 0 ? b_next + (cnt - 1) / k6Batch : b_next;
                    publish_batches(last, cnt > 0 ? cnt - ((cnt - 1) / k6Batch) * k6Batch : 0, k6FlagEnd, X0, Y0, grp);
                    b_next = last + 1;
                    if (lane == 0) {                                         // in shared memory: no registers to spare here
                        S.stat_swept_items += 1;
                        if (cnt > 0) { S.stat_hit_items += 1; S.stat_max_hits = max(S.stat_max_hits, cnt); }
                    }
                }
                if (!publish_item(X0, Y0, grp, false)) { alive = false; break; }
                // ---- advance
                if (sub == 3) { sub = 0; d4 = d4_n; raw_next = claim(); } else ++sub;
                ci = ci_n;
                S_cur = S_n;
                ea = ea_n; eb = eb_n;
            }
            if (lane == 0) S.c_hits = 0x7fffffff;            // nothing left to claim: the store warp may zero-fill at full speed
            // exit: one flagged batch per stager (consumers stop at the first one), one flagged item for the store warp
            if (!*abort_flag) {
                bool ok = true;
                for (int e = 0; e < k6Stagers && ok; ++e) ok = batch_slot_free(b_next + e);
                if (ok) {
                    if (lane == 0) {
                        for (int e = 0; e < k6Stagers; ++e) {
                            const int q = (b_next + e) % k6BatchRing;
                            S.b_n[q] = 0; S.b_flags[q] = k6FlagExit; S.b_x0[q] = 0; S.b_y0[q] = 0; S.b_g[q] = 0;
                        }
                        __threadfence_block();
                        S.pub_batches = b_next + k6Stagers;
                    }
                    __syncwarp();
                }
                publish_item(0, 0, 0, true);
            }
            K6_TOC(t_sw_all, sw0);
            K6_ADD(8, t_sw_all); K6_ADD(9, t_sw_ring); K6_ADD(10, t_sw_item); K6_ADD(11, t_sw_atomic); K6_ADD(22, t_sw_desc); K6_ADD(23, t_sw_loop);
            if (lane == 0 && P.stats) {
                atomicAdd(P.stats + 1, i_pub - 1);                           // consumer items (the exit descriptor is not one)
                atomicAdd(P.stats + 2, S.stat_hit_items);
                atomicAdd(P.stats + 3, b_next);
                atomicMax(P.stats + 4, S.stat_max_hits);
                atomicAdd(P.stats + 5, S.stat_swept_items);
            }
        } else if (role <= k6Stagers) {
            // =========================================================================================== stagers
            // lane = channel.  Every global read of a batch is a cp.async (LDGSTS) straight into the stage: per hit the
            // raw table-offset words of the pre-pass (the consumer adds the tile term), the weights, and the 32 x 32 B of
            // visibilities.  Nothing is computed here on the common path and the stager never waits for its copies: each
            // lane arrives on the batch's mbarrier through cp.async.mbarrier.arrive.noinc, which fires when the lane's
            // copies have landed.  Slow hits (dropped samples, wide spread, ragged last group; rare) are converted with
            // explicit range checks and get zero-filled visibilities where a lane has nothing to contribute.
            // (Per-lane bulk copies, cp.async.bulk = UBLKCP, were measured first: they are issued one lane at a time at
            // ~60 ns each, 6.4 us per 32-hit batch.)
            const int sg = role - 1;                                        // this stager stages batches b = sg, sg + 2, ...
            const u64 pol_last = l2_policy_evict_last();
            (void)pol_last;
            const unsigned zero_geo = (unsigned)(P.n_tu * 4) | ((unsigned)(P.n_tv * 4) << 16);
            const int ncp = P.n_groups * 32;
            long long t_st_pub = 0, t_st_empty = 0, t_st_work = 0, t_st_pre = 0, n_st = 0;
            (void)t_st_pub; (void)t_st_empty; (void)t_st_work; (void)t_st_pre; (void)n_st;
            for (int b = sg;; b += k6Stagers) {
                const int s = b % k6Stages;
                const unsigned st_base = ring_s + (unsigned)s * k6StageBytes;
                const unsigned zs_a = st_base + 16u * lane, geo_a = st_base + k6StageV + 4u * lane, wt_a = geo_a + k6StageGeo;
                const unsigned full_bar = smem_u32(&S.full[s]), empty_bar = smem_u32(&S.empty[s]);
                K6_TIC(q0);
                if (!spin_until_gt(&S.pub_batches, b, abort_flag, K6_ERR_BATCH)) break;
                K6_TOC(t_st_pub, q0);
                __threadfence_block();
                const int q = b % k6BatchRing;
                const int n = S.b_n[q];
                const unsigned flags = S.b_flags[q];
                const int X0 = S.b_x0[q], Y0 = S.b_y0[q], grp = S.b_g[q];
                int row = 0;
                unsigned mask = 0u;
                if (lane < n) { row = S.q_row[q * k6Batch + lane]; mask = S.q_mask[q * k6Batch + lane]; }
                __syncwarp();
                const int use = b / k6Stages;                                // this stage's use number
                K6_TIC(q1);
                if (!mbar_wait(empty_bar, (unsigned)((use & 1) ^ 1), abort_flag, K6_ERR_EMPTY)) break;
                K6_TOC(t_st_empty, q1);
                K6_TIC(q2);
                const int c0 = grp * 32;
                const bool cvalid = c0 + lane < P.n_chan;                    // the last group may be ragged
                const int cc = cvalid ? c0 + lane : P.n_chan - 1;            // a valid address for every lane
                const unsigned slow_m = __ballot_sync(full, lane < n && (((mask >> 16) & 1u) || c0 + 32 > P.n_chan));
                const unsigned tile_c = (unsigned)(4 * (X0 - k6Bias)) + ((unsigned)(4 * (Y0 - k6Bias)) << 16);
                if (lane < k6Batch) S.st_mask[s][lane] = lane < n ? (mask & 0xffffu) : 0u;
                if (lane == 0) { S.st_n[s] = n; S.st_flags[s] = flags; S.st_tile[s] = tile_c; }
                for (int hh = 0; hh < n; ++hh) {
                    const int r = __shfl_sync(full, row, hh);
                    if ((slow_m >> hh) & 1u) continue;                       // uniform
                    if (HAS_W)
                        asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(wt_a + 128u * (unsigned)hh), "l"(P.weights + (size_t)r * P.n_chan + cc) : "memory");
                    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(geo_a + 128u * (unsigned)hh), "l"(P.pre + (size_t)r * ncp + c0 + lane) : "memory");
#ifndef K6_ABLATE_LOAD
                    const float* src = P.vis + ((size_t)r * P.n_chan + cc) * 8;
#if defined(K6_NO_L2_HINTS) || !defined(K6_VIS_EVICT_LAST)
                    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(zs_a + 1024u * (unsigned)hh), "l"(src) : "memory");
                    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(zs_a + 1024u * (unsigned)hh + 512u), "l"(src + 4) : "memory");
#else
                    asm volatile("cp.async.cg.shared.global.L2::cache_hint [%0], [%1], 16, %2;" ::"r"(zs_a + 1024u * (unsigned)hh), "l"(src), "l"(pol_last) : "memory");
                    asm volatile("cp.async.cg.shared.global.L2::cache_hint [%0], [%1], 16, %2;" ::"r"(zs_a + 1024u * (unsigned)hh + 512u), "l"(src + 4), "l"(pol_last) : "memory");
#endif
#endif
                }
                for (unsigned sm_ = slow_m; sm_ != 0u; sm_ &= sm_ - 1u) {   // slow hits: packed (origin, table row) words, range-checked here
                    const int hh = __ffs(sm_) - 1;
                    const int r = __shfl_sync(full, row, hh);
                    const unsigned w32 = __ldg(P.pre + (size_t)r * ncp + c0 + lane);
                    unsigned geo = zero_geo;
                    if (w32 != k6Invalid) {
                        const int ou = (int)(w32 & 0x7ffu), ru = (int)((w32 >> 11) & 31u);
                        const int ov = (int)((w32 >> 16) & 0x7ffu), rv = (int)(w32 >> 27);
                        const int tu_ = k6PadU + X0 - ou, tv_ = k6PadV + Y0 - ov;
                        const unsigned iu_ = (unsigned)(W - 1 + ou - X0), iv_ = (unsigned)(W - 1 + ov - Y0);
                        if (iu_ < (unsigned)(k6TileX + W - 1) && iv_ < (unsigned)(k6TileY + W - 1)) {
                            const int su = tu_ & 3, sv = tv_ & 1;
                            const int offu = ru * P.rlu + tu_ + su * (O1 * P.rlu - 1);
                            const int offv = rv * P.rlv + tv_ + sv * (O1 * P.rlv - 1);
                            geo = (unsigned)(offu * 4) | ((unsigned)(offv * 4) << 16);
                        }
                    }
                    geo -= tile_c;                                           // the consumer adds the tile term to every word
                    asm volatile("st.shared.u32 [%0], %1;" ::"r"(geo_a + 128u * (unsigned)hh), "r"(geo) : "memory");
                    const float* src = P.vis + ((size_t)r * P.n_chan + cc) * 8;
                    const unsigned sz = (cvalid && w32 != k6Invalid) ? 16u : 0u;   // zero-filled where the lane has no sample (R11)
                    if (HAS_W)                                               // the weight as well: a flagged NaN must not reach a product
                        asm volatile("cp.async.ca.shared.global [%0], [%1], 4, %2;" ::"r"(wt_a + 128u * (unsigned)hh), "l"(P.weights + (size_t)r * P.n_chan + cc), "r"(sz >> 2) : "memory");
                    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(zs_a + 1024u * (unsigned)hh), "l"(src), "r"(sz) : "memory");
                    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(zs_a + 1024u * (unsigned)hh + 512u), "l"(src + 4), "r"(sz) : "memory");
                }
                // the batch is complete when all 32 lanes' copies have landed (noinc arrivals) and the meta data are written
                asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(full_bar) : "memory");
                __syncwarp();
                if (lane == 0) {
                    mbar_arrive(full_bar);
                    __threadfence_block();
                    S.done_batches[sg] = b / k6Stagers + 1;                  // queue segment and descriptor of batch b are free again
                }
                K6_TOC(t_st_work, q2);
#ifdef K6_TIMING
                ++n_st;
#endif
                if (flags & k6FlagExit) break;
            }
            asm volatile("cp.async.wait_all;" ::: "memory");
            K6_ADD(12, t_st_pub); K6_ADD(13, t_st_empty); K6_ADD(14, t_st_work); K6_ADD(15, n_st); K6_ADD(21, t_st_pre);
        } else {
            // =========================================================================================== store warp
            // One thread.  Consumer items come in order: the tensor-map store of each of their four block rows is issued
            // as soon as that row's four warps have staged it, and the stage is handed back as soon as the TMA engine has
            // read it (it is single-buffered: its consumers need it at the end of their next item).  Items nothing reaches
            // are zero-filled from the zero buffer at low priority, four 4 KB boxes at a time, between looks at the rows.
            // (Plain st.global zero-fill from this one warp was measured at 4 B / clock - latency-throttled.)
            if (lane == 0) {
                const unsigned wo0 = smem_u32(base + L.wo), zero_s = smem_u32(base + L.zero);
                const u64 pol_first = l2_policy_evict_first();
                int ci = 0, zc = 0;                                          // consumer item, 4-store chunk of the current zero item
                // zero items are claimed 16 at a time from the list of chan_order_kernel; the claim of the next chunk is in
                // flight while this one is stored (one exposed L2 round trip per 16 items of ~3 us each)
                const int n_z = __ldg(P.n_cz + 1);
                int z_cur = -1, z_k = 0, z_n = 0, zX0 = 0, zY0 = 0, zc0 = 0, z_pos = 0;
                const long long n_hits = max(__ldg(P.n_hits), 1);
                const long long z_lead = n_hits * K6_ZERO_LEAD_PCT / 100 + 64;
                int z_base_next = atomicAdd(P.zcounter, k6ZeroChunk);
                int zb_cur = 0;
                auto z_advance = [&]() {
                    if (z_k >= z_n) {
                        const int zb = z_base_next;
                        if (zb >= n_z) { z_cur = -1; return; }           // claims only grow: the list is exhausted for good
                        z_n = min(k6ZeroChunk, n_z - zb);
                        zb_cur = zb;
                        const int4* src = reinterpret_cast<const int4*>(P.z_list + zb);   // 64 B aligned; the list is padded
#pragma unroll
                        for (int q = 0; q < k6ZeroChunk / 4; ++q) reinterpret_cast<int4*>(S.z_ids)[q] = __ldg(src + q);
                        z_base_next = atomicAdd(P.zcounter, k6ZeroChunk);
                        z_k = 0;
                    }
                    z_pos = zb_cur + z_k;
                    z_cur = S.z_ids[z_k++];
                    int tx, ty, grp;
                    k6_item_decode(P, z_cur, tx, ty, grp);
                    zX0 = tx * k6TileX; zY0 = ty * k6TileY; zc0 = grp * 32;
                };
                if (!P.accumulate) z_advance();                          // accumulate-into leaves the cells nothing reaches alone
                unsigned remaining = 0xfu;                                   // block rows of consumer item ci still to store
                long long t_so_rel = 0, t_so_idle = 0, t_so_zero = 0, t_so_all = 0;
                (void)t_so_rel; (void)t_so_idle; (void)t_so_zero; (void)t_so_all;
                K6_TIC(so0);
                long long idle_t0 = 0;
                bool idle = false;
                for (;;) {
                    bool progress = false;
                    if (S.pub_c > ci) {
                        __threadfence_block();
                        const unsigned word = S.c_item[ci % k6ItemRing];
                        if (word == k6ExitItem) {
                            if (z_cur < 0) break;                            // the zero list is exhausted as well (claims only grow)
                        } else {
                            const int X0 = (int)(word & 1023u) * k6TileX, Y0 = (int)((word >> 10) & 1023u) * k6TileY, c0 = (int)(word >> 20) * 32;
#pragma unroll
                            for (int r = 0; r < 4; ++r) {
                                // rows r and r + 2 share a slot and take turns: row r + 2 is looked at once row r is stored
                                const unsigned par = (unsigned)((2 * ci + (r >> 1)) & 1);
                                if (((remaining >> r) & 1u) && (r < 2 || !((remaining >> (r - 2)) & 1u)) && mbar_try(smem_u32(&S.wo_full[r & 1]), par)) {
#ifndef K6_ABLATE_STORE
                                    if (Y0 + 2 * r < N) {
                                        if (P.accumulate) tma_reduce_add4(&map_acc, wo0 + 32768u * (r & 1), 2 * X0, c0, Y0 + 2 * r, 0);
                                        else tma_store4(&map_out, wo0 + 32768u * (r & 1), X0, c0, Y0 + 2 * r, 0, pol_first);
                                    }
#endif
                                    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
                                    K6_TIC(s0);
                                    asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
                                    K6_TOC(t_so_rel, s0);
                                    mbar_arrive(smem_u32(&S.wo_empty[r]));
                                    remaining &= ~(1u << r);
                                    progress = true;
                                }
                            }
                            if (remaining == 0u) { ++ci; S.done_c = ci; remaining = 0xfu; }
                        }
                    }
                    // Zero-fill is paced by the progress of the consumer items (both lists are global and claimed in order): the
                    // share of the zero list that is done stays within K6_ZERO_LEAD_PCT of the share of all HITS that lie before
                    // the item the sweeper is on (c_desc.w) - the work measure, so the zeros flow while the consumers are busy.  Unpaced, every SM zero-fills flat out at the start of the kernel and the write
                    // stream starves the visibility loads of the dense tiles (measured: 8.2 - 8.6 ms against 7.9).
                    if (z_cur >= 0 && (long long)z_pos * n_hits <= ((long long)S.c_hits + z_lead) * n_z) {
                        K6_TIC(s2);
                        // one box of [v 4][chan 32][16 cells] per look, and never more than K6_ZERO_INFLIGHT + 1 of them queued in
                        // the TMA engine: a consumer row that becomes ready must not wait behind a long run of zero boxes
#ifndef K6_ZERO_INFLIGHT
#define K6_ZERO_INFLIGHT 1
#endif
                        asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(K6_ZERO_INFLIGHT) : "memory");
                        const int zpol = zc / (k6TileY / k6ZeroV), zv = (zc % (k6TileY / k6ZeroV)) * k6ZeroV;
#ifndef K6_ABLATE_STORE
                        if (zY0 + zv < N) tma_store4(&map_zero, zero_s, zX0, zc0, zY0 + zv, zpol, pol_first);
#endif
                        asm volatile("cp.async.bulk.commit_group;" ::: "memory");
                        if (++zc == 4 * (k6TileY / k6ZeroV)) { zc = 0; z_advance(); }
                        progress = true;
                        K6_TOC(t_so_zero, s2);
                    }
                    if (progress) {
#ifdef K6_TIMING
                        if (idle) t_so_idle += clock64() - idle_t0;
#endif
                        idle = false;
                    } else {
                        if (!idle) { idle_t0 = clock64(); idle = true; }
                        if (*abort_flag) break;
                        if (clock64() - idle_t0 > k6SpinLimit) { *abort_flag = K6_ERR_WOFULL; break; }
                    }
                }
                asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");   // every store has landed before the CTA exits
                K6_TOC(t_so_all, so0);
                K6_ADD(16, t_so_all); K6_ADD(17, t_so_rel); K6_ADD(18, t_so_idle); K6_ADD(20, t_so_zero);
            }
        }
    }
    __syncthreads();
    if (tid == 0 && S.abort && P.stats) atomicMax(P.stats, S.abort);
}

// ------------------------------------------------------------------------------------------------ host side
static void chanws_table_geometry(const GridGeom& g, K6Params& P) {
    P.rlu = (k6PadU + g.W + 15 + k6Drift + 3) & ~3;     // pad + W + (tile - 1) + drift more taps to the right, multiple of 4
    P.rlv = (k6PadV + g.W + 7 + k6Drift + 1) & ~1;      // pad + W + (tile - 1) + drift, multiple of 2
    P.n_tu = 4 * (g.O + 1) * P.rlu;
    P.n_tv = 2 * (g.O + 1) * P.rlv;
}

long long chanws_items(const Plan* p, int n_chan) {
    const long long ntx = (p->geom.N + k6TileX - 1) / k6TileX, nty = (p->geom.N + k6TileY - 1) / k6TileY;
    return ntx * nty * ((n_chan + 31) / 32);
}

bool chanws_supported(const Plan* p, int n_chan) {
    if (n_chan < 1) return false;
    if (p->geom.N > 2048 || p->geom.O > 30) return false;                    // 11 + 5 bits per axis in the packed index
    K6Params P;
    chanws_table_geometry(p->geom, P);
    if ((P.n_tu + k6ZeroFloats) * 4 > 65535 || (P.n_tv + k6ZeroFloats) * 4 > 65535) return false;   // geo packs 16-bit byte offsets
    return k6_layout(P.n_tu, P.n_tv).total <= 227 * 1024;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn encode_tiled_fn() {
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess)
            return nullptr;
        fn = reinterpret_cast<EncodeTiledFn>(p);
    }
    return fn;
}

// grid_out [n_chan][4][N][N] complex64 seen as a 4-D tensor of 8-byte elements with dimension order (u, channel, v, pol)
static bool make_grid_map(CUtensorMap* map, float* grid, int N, int n_chan, int box_v, int box_pol, bool swizzle,
                          bool as_floats = false) {
    EncodeTiledFn enc = encode_tiled_fn();
    if (!enc) { set_error("cuTensorMapEncodeTiled is not available from the driver"); return false; }
    // as_floats: the same memory as 4-byte elements (u is 2 N floats long, the box 32 floats wide) - what a reduce-add needs
    const cuuint64_t dims[4] = {(cuuint64_t)(as_floats ? 2 * N : N), (cuuint64_t)n_chan, (cuuint64_t)N, 4};
    const cuuint64_t strides[3] = {(cuuint64_t)4 * N * N * 8, (cuuint64_t)N * 8, (cuuint64_t)N * N * 8};
    const cuuint32_t box[4] = {as_floats ? 32u : 16u, 32, (cuuint32_t)box_v, (cuuint32_t)box_pol};
    const cuuint32_t es[4] = {1, 1, 1, 1};
    const CUresult r = enc(map, as_floats ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_UINT64, 4, grid, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                           swizzle ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { set_error("cuTensorMapEncodeTiled failed (CUresult " + std::to_string((int)r) + ")"); return false; }
    return true;
}

bool launch_chanws(Plan* p, const float* vis, const float* w, long long n_vis, int n_chan, float* grid,
                   const int* dispatch, cudaStream_t st) {
    if (!chanws_supported(p, n_chan)) { set_error("design CHANWS does not support this grid / kernel table size"); return false; }
    Workspace& ws = p->ws;
    K6Params P;
    P.g = p->geom;
    chanws_table_geometry(p->geom, P);
    P.group = (const double4*)ws.d_group;
    P.bucket_start = ws.d_bucket_count;
    P.perm = ws.d_perm;
    P.pre = ws.d_pre;
    P.bb = (const ushort4*)ws.d_bb;
    P.pool_cap = ws.pool_cap;
    P.list_cnt = ws.d_list_cnt;
    P.list_off = ws.d_list_off;
    P.c_desc = (const int4*)ws.d_c_desc;
    P.z_list = ws.d_z_list;
    P.n_cz = ws.d_misc + 14;
    P.n_hits = ws.d_misc + 11;
    P.zcounter = ws.d_misc + 3;
    P.lists = (const uint2*)ws.d_lists;
    P.counter = ws.d_misc + 2;
    P.stats = ws.d_misc + 4;
    P.dispatch = dispatch;
    P.dispatch_want = 1;
    P.vis = vis;
    P.weights = w;
    P.table = p->d_table;
    P.grid = grid;
    P.n_vis = (int)n_vis;
    P.n_chan = n_chan;
    P.n_groups = (n_chan + 31) / 32;
    P.nb = (p->geom.N + kBucketCells - 1) / kBucketCells;
    P.ntx = (p->geom.N + k6TileX - 1) / k6TileX;
    P.nty = (p->geom.N + k6TileY - 1) / k6TileY;
    P.n_items = (long long)P.ntx * P.nty * P.n_groups;
    if (P.n_items >= 0x7fffffffLL) { set_error("design CHANWS: too many work items"); return false; }
    CUtensorMap map_out, map_zero, map_acc;
    P.accumulate = p->accumulate ? 1 : 0;
    if (!make_grid_map(&map_out, grid, p->geom.N, n_chan, 2, 4, true)) return false;
    if (!make_grid_map(&map_zero, grid, p->geom.N, n_chan, k6ZeroV, 1, false)) return false;
    if (!make_grid_map(&map_acc, grid, p->geom.N, n_chan, 2, 4, true, true)) return false;

    long long iblocks = (n_vis + 7) / 8;                                      // one warp per sorted row at a time
    if (iblocks > (long long)p->sm_count * 8) iblocks = (long long)p->sm_count * 8;
    if (iblocks < 1) iblocks = 1;
    chan_index_kernel<<<(unsigned)iblocks, 256, 0, st>>>(p->geom, (const double4*)ws.d_row_sorted, ws.d_scale, (int)n_vis, n_chan,
                                                         P.n_groups, P.rlu, P.rlv, ws.d_pre, (ushort4*)ws.d_bb, dispatch, 1);
    {
        long long lblocks = (P.n_items + 7) / 8;
        if (lblocks > (long long)p->sm_count * 32) lblocks = (long long)p->sm_count * 32;
        chan_list_kernel<<<(unsigned)lblocks, 256, 0, st>>>(P, ws.d_list_cnt, ws.d_list_off, (uint2*)ws.d_lists,
                                                            reinterpret_cast<unsigned long long*>(ws.d_misc + 12));
        int per_block = (int)(((P.n_items + k6OrderBlocksMax - 1) / k6OrderBlocksMax + 1023) / 1024) * 1024;
        const int oblocks = (int)((P.n_items + per_block - 1) / per_block);
        chan_order_kernel<<<oblocks, 1024, 0, st>>>(ws.d_list_cnt, ws.d_list_off, (int)P.n_items, per_block, (int4*)ws.d_c_desc,
                                                    ws.d_z_list, ws.d_misc + 14, ws.d_misc + 11, (P.n_groups - 1) * P.ntx * P.nty, ws.d_misc + kMiscTailStart,
                                                    ws.d_misc + kMiscOrderState, dispatch, 1);
        if (!cuda_ok(cudaFuncSetAttribute(chan_tail_sort_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, k6TailMax * 24), "tail sort smem attribute"))
            return false;
        chan_tail_sort_kernel<<<1, 1024, k6TailMax * 24, st>>>((int4*)ws.d_c_desc, ws.d_misc + 14, ws.d_misc + kMiscTailStart, dispatch, 1);
    }
    const size_t smem = k6_layout(P.n_tu, P.n_tv).total;
    auto kern = w ? chanws_kernel<true> : chanws_kernel<false>;
    if (!cuda_ok(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem), "chanws smem attribute"))
        return false;
    long long blocks = p->sm_count;
    if (blocks > P.n_items) blocks = P.n_items;
    kern<<<(unsigned)blocks, k6Threads, smem, st>>>(P, map_out, map_zero, map_acc);
    p->last_launches += 5;
    return cuda_ok(cudaGetLastError(), "chanws_kernel");
}

}  // namespace mwa
