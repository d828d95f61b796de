// k_bin.cu - a3: counting sort of the n_vis baseline rows by uv bucket (hard part 1).
//
// u_lambda = u_m * nu / c is a pure radial scaling, so the rows are binned ONCE per call, at the largest
// channel scale s_ref of the call, into kBucketCells-wide buckets.  A (tile, channel) work item of the
// gridder back-projects its tile (plus the stamp halo) to the reference scale, walks the few buckets
// that overlap it, and decides membership with the exact index function; the buckets only have to be
// conservative.  n_vis items are sorted, not n_vis * n_chan.
//
// Launches: the two memsets, scale_kernel (k_basic.cu), then - each as a programmatic dependent of the one before (plan.h:
// launch_dependent; every kernel starts with pdl_wait / pdl_release) - bin_count, bin_scan, bin_scatter, bin_order, bin_order_large, tile_weight, tile_order_scan,
// tile_order_scatter.  Small calls (<= 4096 rows) do all of it, and a1, in the single CTA of bin_small_kernel.
#include "plan.h"
#include "scale.cuh"

namespace mwa {

__device__ __forceinline__ int bucket_coord(double metres, double s_ref, double inv_du, int N, int nb) {
    const double cx = metres * s_ref * inv_du + (double)(N / 2);     // cells from the low grid edge
    if (!(cx > 0.0)) return 0;                                        // also NaN
    const double b = floor(cx * (1.0 / kBucketCells));
    return b >= (double)(nb - 1) ? nb - 1 : (int)b;
}

__global__ void bin_count_kernel(GridGeom g, const double2* __restrict__ uv, const double* __restrict__ s_ref_p,
                                 int n_vis, int nb, int* __restrict__ count) {
    pdl_wait();                                         // chain of dependent launches (plan.h)
    pdl_release();
    const double s_ref = *s_ref_p;
    for (int n = blockIdx.x * blockDim.x + threadIdx.x; n < n_vis; n += gridDim.x * blockDim.x) {
        const double2 p = uv[n];
        const int bx = bucket_coord(p.x, s_ref, g.inv_du, g.N, nb);
        const int by = bucket_coord(p.y, s_ref, g.inv_du, g.N, nb);
        atomicAdd(&count[by * nb + bx], 1);
    }
}

// Exclusive scan of count[0..n] in place (count[n] receives the total).  A block of 1024 threads takes 4096 consecutive
// entries, publishes its sum in blk_state (zeroed by the call's memset; flag bit 30) and adds up the sums of the blocks
// before it - they were scheduled before it, so the wait cannot deadlock (the one-level decoupled scan of
// chan_order_kernel; a single block needed 15 - 60 us for the 16 K - 262 K buckets of C4 - C5).
constexpr int kScanPerBlock = 4096;
constexpr int kScanFlag = 1 << 30;

__global__ void __launch_bounds__(1024)
bin_scan_kernel(int* __restrict__ count, int n, int* __restrict__ cursor, volatile int* blk_state) {
    pdl_wait();                                         // chain of dependent launches (plan.h)
    pdl_release();
    __shared__ int warp_sum[32];
    __shared__ int prefix_s;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, b = blockIdx.x;
    const int i0 = b * kScanPerBlock + threadIdx.x * 4;
    int v[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) v[k] = (i0 + k < n) ? count[i0 + k] : 0;
    const int tsum = v[0] + v[1] + v[2] + v[3];
    int inc = tsum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) warp_sum[wid] = inc;
    __syncthreads();
    if (wid == 0) {
        int ws = warp_sum[lane];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, ws, o);
            if (lane >= o) ws += t;
        }
        warp_sum[lane] = ws;                     // inclusive over warps
        const int total = __shfl_sync(0xffffffffu, ws, 31);
        if (lane == 0) blk_state[b] = total | kScanFlag;
        int sum = 0;
        for (int j0 = 0; j0 < b; j0 += 32) {
            const int j = j0 + lane;
            int t = 0;
            if (j < b) {
                do { t = blk_state[j]; } while (!(t & kScanFlag));
                t &= ~kScanFlag;
            }
            sum += t;
        }
        sum = __reduce_add_sync(0xffffffffu, sum);
        if (lane == 0) {
            prefix_s = sum;
            if (b == (int)gridDim.x - 1) count[n] = sum + total;
        }
    }
    __syncthreads();
    int excl = prefix_s + (wid > 0 ? warp_sum[wid - 1] : 0) + inc - tsum;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        if (i0 + k < n) { count[i0 + k] = excl; cursor[i0 + k] = excl; }
        excl += v[k];
    }
}

__global__ void bin_scatter_kernel(GridGeom g, const double2* __restrict__ uv, const double* __restrict__ s_ref_p,
                                   int n_vis, int nb, int* __restrict__ cursor, int* __restrict__ perm_tmp) {
    pdl_wait();                                         // chain of dependent launches (plan.h)
    pdl_release();
    const double s_ref = *s_ref_p;
    for (int n = blockIdx.x * blockDim.x + threadIdx.x; n < n_vis; n += gridDim.x * blockDim.x) {
        const double2 p = uv[n];
        const int bx = bucket_coord(p.x, s_ref, g.inv_du, g.N, nb);
        const int by = bucket_coord(p.y, s_ref, g.inv_du, g.N, nb);
        perm_tmp[atomicAdd(&cursor[by * nb + bx], 1)] = n;            // order inside a bucket: whatever the atomics gave
    }
}

// One warp per bucket puts the bucket's rows in ascending row order (rank = number of smaller row ids; buckets hold
// ~8 rows on average, a few hundred in the core) and writes the sorted copies.  With this the bucket-sorted order is a
// pure function of the input, so K3c and K5 - which add the taps of a cell in list order, with no atomics - give
// bit-identical grids from run to run.
// A bucket of more than kOrderWarpMax rows (the core of a dense array; or a degenerate input: a compact array, a coarse
// du, many rows at uv = 0) is not ranked here - k^2 / 32 steps per lane make one warp the critical path of the call -
// but put on a list for bin_order_large_kernel, which gives it a whole block.
constexpr int kOrderWarpMax = 256;                     // buckets up to this many rows are ranked by one warp, from shared memory
constexpr int kOrderStage = kOrderWarpMax;
constexpr int kOrderBlockRank = 2048;                  // bin_order_large_kernel: up to this many rows by counting, beyond by bitonic sort
constexpr int kBigListCap = 1023;                      // buckets beyond the list are ranked by their warp of bin_order_kernel

__global__ void bin_order_kernel(const double2* __restrict__ uv, const int* __restrict__ bucket_start, int n_buckets,
                                 const int* __restrict__ perm_tmp, int* __restrict__ perm,
                                 double2* __restrict__ uv_sorted, double4* __restrict__ row_sorted, int* __restrict__ big_list) {
    pdl_wait();                                         // chain of dependent launches (plan.h)
    pdl_release();
    __shared__ int s_stage[8][kOrderStage];                // blocks of 256 threads
    const int lane = threadIdx.x & 31;
    int* stage = s_stage[(threadIdx.x >> 5) & 7];
    const int warps = (gridDim.x * blockDim.x) >> 5;
    for (int b = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; b < n_buckets; b += warps) {
        const int k0 = bucket_start[b], k1 = bucket_start[b + 1];
        if (k1 - k0 > kOrderWarpMax) {
            int slot = 0;
            if (lane == 0) {
                slot = atomicAdd(big_list, 1);
                if (slot < kBigListCap) big_list[1 + slot] = b;
            }
            if (__shfl_sync(0xffffffffu, slot, 0) < kBigListCap) continue;
            // the list is full (more than 1023 such buckets): this warp ranks the bucket itself, slowly, below
        }
        const int k = k1 - k0;
        if (k > 32 && k <= kOrderStage) {
            // the dense buckets of a core (hundreds of rows) are what this kernel's time is made of: the bucket is staged in
            // shared memory and a lane ranks four of its rows per pass over it (one broadcast LDS per four compares)
            __syncwarp();
            for (int i = lane; i < k; i += 32) stage[i] = perm_tmp[k0 + i];
            __syncwarp();
            for (int i0 = lane; i0 < k; i0 += 128) {
                int row[4], rank[4] = {0, 0, 0, 0};
#pragma unroll
                for (int t = 0; t < 4; ++t) row[t] = i0 + 32 * t < k ? stage[i0 + 32 * t] : 0x7fffffff;
                for (int j = 0; j < k; ++j) {
                    const int v = stage[j];
#pragma unroll
                    for (int t = 0; t < 4; ++t) rank[t] += v < row[t];
                }
#pragma unroll
                for (int t = 0; t < 4; ++t) {
                    if (i0 + 32 * t < k) {
                        const double2 p = uv[row[t]];
                        perm[k0 + rank[t]] = row[t];
                        uv_sorted[k0 + rank[t]] = p;
                        row_sorted[k0 + rank[t]] = make_double4(p.x, p.y, (double)row[t], 0.0);
                    }
                }
            }
            continue;
        }
        for (int i = k0 + lane; i < k1; i += 32) {
            const int row = perm_tmp[i];
            int rank = 0;
            for (int j = k0; j < k1; ++j) rank += perm_tmp[j] < row;
            const double2 p = uv[row];
            perm[k0 + rank] = row;
            uv_sorted[k0 + rank] = p;
            row_sorted[k0 + rank] = make_double4(p.x, p.y, (double)row, 0.0);      // K5: uv and row id in one 32 B record
        }
    }
}

// The big buckets: one block each sorts the bucket's row ids ascending in place - a bitonic network in its all-ascending
// form (first step of a merge mirrors inside the block of size k, the rest are half-cleaners), so a length that is not a
// power of two needs no padding: a partner index beyond the end stands for +infinity, which is already in place - and
// writes the sorted copies.  O(k log^2 k): 1 M rows in ~2 ms.  Returns at once when the list is empty (every normal call).
__global__ void __launch_bounds__(1024)
bin_order_large_kernel(const double2* __restrict__ uv, const int* __restrict__ bucket_start, int* __restrict__ perm_tmp,
                       int* __restrict__ perm, double2* __restrict__ uv_sorted, double4* __restrict__ row_sorted,
                       const int* __restrict__ big_list) {
    pdl_wait();                                         // chain of dependent launches (plan.h)
    pdl_release();
    __shared__ int s_rows[kOrderBlockRank];
    const int n_big = min(big_list[0], kBigListCap);
    for (int q = blockIdx.x; q < n_big; q += gridDim.x) {
        const int b = big_list[1 + q];
        const int k0 = bucket_start[b], n = bucket_start[b + 1] - k0;
        int* a = perm_tmp + k0;
        if (n <= kOrderBlockRank) {                          // the dense buckets of a core: rank by counting, from shared memory
            for (int i = threadIdx.x; i < n; i += 1024) s_rows[i] = a[i];
            __syncthreads();
            for (int i0 = threadIdx.x; i0 < n; i0 += 2048) {
                const int r0 = s_rows[i0], r1 = i0 + 1024 < n ? s_rows[i0 + 1024] : 0x7fffffff;
                int rank0 = 0, rank1 = 0;
                for (int j = 0; j < n; ++j) {
                    const int v = s_rows[j];
                    rank0 += v < r0;
                    rank1 += v < r1;
                }
                {
                    const double2 p = uv[r0];
                    perm[k0 + rank0] = r0;
                    uv_sorted[k0 + rank0] = p;
                    row_sorted[k0 + rank0] = make_double4(p.x, p.y, (double)r0, 0.0);
                }
                if (i0 + 1024 < n) {
                    const double2 p = uv[r1];
                    perm[k0 + rank1] = r1;
                    uv_sorted[k0 + rank1] = p;
                    row_sorted[k0 + rank1] = make_double4(p.x, p.y, (double)r1, 0.0);
                }
            }
            __syncthreads();
            continue;
        }
        for (int k = 2; (k >> 1) < n; k <<= 1) {
            for (int i = threadIdx.x; i < n; i += 1024) {            // mirror step
                const int j = i ^ (k - 1);
                if (j > i && j < n) { const int x = a[i], y = a[j]; if (x > y) { a[i] = y; a[j] = x; } }
            }
            __syncthreads();
            for (int d = k >> 2; d > 0; d >>= 1) {                   // half-cleaners
                for (int i = threadIdx.x; i < n; i += 1024) {
                    const int j = i ^ d;
                    if (j > i && j < n) { const int x = a[i], y = a[j]; if (x > y) { a[i] = y; a[j] = x; } }
                }
                __syncthreads();
            }
        }
        for (int i = threadIdx.x; i < n; i += 1024) {
            const int row = a[i];
            const double2 p = uv[row];
            perm[k0 + i] = row;
            uv_sorted[k0 + i] = p;
            row_sorted[k0 + i] = make_double4(p.x, p.y, (double)row, 0.0);
        }
        __syncthreads();
    }
}

// Tile weights (rows whose reference-scale bucket lies under the tile) and a heaviest-first tile order by a
// counting sort on the clipped weight.  Only a scheduling heuristic: any order gives the same grid.

__global__ void tile_weight_kernel(const int* __restrict__ bucket_start, int nb, int nt, int* __restrict__ weight,
                                   int* __restrict__ hist) {
    pdl_wait();                                         // chain of dependent launches (plan.h)
    pdl_release();
    const int per = kTile / kBucketCells, lane = threadIdx.x & 31;
    // a warp walks 32 consecutive tiles per pass (the loop bound is uniform in the warp: the warp-wide votes below are safe)
    for (int t0 = (blockIdx.x * blockDim.x + threadIdx.x) & ~31; t0 < nt * nt; t0 += gridDim.x * blockDim.x) {
        const int t = t0 + lane;
        const bool valid = t < nt * nt;
        const unsigned act = __ballot_sync(0xffffffffu, valid);
        if (!valid) continue;
        const int ty = t / nt, tx = t - ty * nt;
        int w = 0;
        for (int dy = 0; dy < per; ++dy) {
            const int by = ty * per + dy;
            if (by >= nb) break;
            const int b0 = by * nb + tx * per;
            const int b1 = by * nb + min(nb, tx * per + per);
            if (b0 < b1) w += bucket_start[b1] - bucket_start[b0];
        }
        weight[t] = w;
        // descending; one atomic per distinct bin of the warp (most tiles of a sparse grid are empty: one bin for all of them)
        const int bin = kWeightBins - 1 - min(w, kWeightBins - 1);
        const unsigned same = __match_any_sync(act, bin);
        if (__ffs(same) - 1 == lane) atomicAdd(&hist[bin], __popc(same));
    }
}

__global__ void tile_order_scan_kernel(int* __restrict__ hist) {   // one block of kWeightBins threads
    pdl_wait();                                         // chain of dependent launches (plan.h)
    pdl_release();
    __shared__ int s[kWeightBins];
    s[threadIdx.x] = hist[threadIdx.x];
    __syncthreads();
    for (int o = 1; o < kWeightBins; o <<= 1) {
        const int t = threadIdx.x >= o ? s[threadIdx.x - o] : 0;
        __syncthreads();
        s[threadIdx.x] += t;
        __syncthreads();
    }
    hist[threadIdx.x] = s[threadIdx.x] - hist[threadIdx.x];         // exclusive
}

__global__ void tile_order_scatter_kernel(const int* __restrict__ weight, int n_tiles, int* __restrict__ hist,
                                          int* __restrict__ order) {
    pdl_wait();                                         // chain of dependent launches (plan.h)
    pdl_release();
    const int lane = threadIdx.x & 31;
    for (int t0 = (blockIdx.x * blockDim.x + threadIdx.x) & ~31; t0 < n_tiles; t0 += gridDim.x * blockDim.x) {
        const int t = t0 + lane;
        const bool valid = t < n_tiles;
        const unsigned act = __ballot_sync(0xffffffffu, valid);
        if (!valid) continue;
        const int bin = kWeightBins - 1 - min(weight[t], kWeightBins - 1);
        const unsigned same = __match_any_sync(act, bin);                 // the lanes of one bin take consecutive places
        const int leader = __ffs(same) - 1;
        int pos = 0;
        if (lane == leader) pos = atomicAdd(&hist[bin], __popc(same));
        pos = __shfl_sync(same, pos, leader) + __popc(same & ((1u << lane) - 1u));
        order[pos] = t;
    }
}

// ---------------------------------------------------------------- small problems: the whole of a3 in one CTA
// C1-sized calls (<= 4096 rows, <= 2048 buckets, <= 1024 tiles) are launch-bound: seven binning kernels and a memset
// for a problem whose roofline is below a microsecond.  One block of 1024 threads does the same steps in shared memory -
// histogram, scan, scatter, ascending row order inside every bucket, tile weights and the heaviest-first tile order - and
// writes the same arrays (bucket_start, perm, uv_sorted, row_sorted, tile_weight, tile_order) with the same contents,
// except that equal-weight tiles are ordered by index here (the multi-kernel path orders them as its atomics fall).
// With freqs != null the block first does a1 (scale.cuh) and clears the call's counters itself: the whole pre-pass of a
// small call is then ONE launch instead of scale_kernel + memset + this kernel (launch_small_prepass).
constexpr int kSmallRows = 4096, kSmallBuckets = 2048, kSmallTiles = 1024;   // 36 KB of static shared memory

__global__ void __launch_bounds__(1024)
bin_small_kernel(GridGeom g, const double2* __restrict__ uv, const double* __restrict__ s_ref_p, int n_vis, int nb, int nt,
                 int* __restrict__ bucket_start, int* __restrict__ perm, double2* __restrict__ uv_sorted,
                 double4* __restrict__ row_sorted, int* __restrict__ tile_weight, int* __restrict__ tile_order,
                 const double* __restrict__ freqs, int n_chan, int chan_ok, double* __restrict__ scale,
                 double* __restrict__ scale_ref, int* __restrict__ dispatch, double4* __restrict__ group, int* __restrict__ misc) {
    __shared__ int s_start[kSmallBuckets + 1];      // counts, then exclusive starts
    __shared__ int s_cursor[kSmallBuckets];
    __shared__ unsigned short s_tmp[kSmallRows];    // rows in bucket order, arbitrary inside a bucket
    __shared__ unsigned short s_bkt[kSmallRows];    // bucket of row n
    __shared__ int s_warp[32];
    __shared__ int s_tw[kSmallTiles];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int n_buckets = nb * nb, n_tiles = nt * nt;
    double s_ref;
    if (freqs != nullptr) {                         // fused pre-pass: a1 and the memset of the counters
        // a gridder launched with programmatic stream serialisation may start its prologue now (it waits for this grid's
        // completion before it reads anything written here); without such a launch the instruction does nothing
        asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
        s_ref = scale_block(freqs, n_chan, g.N / 2, chan_ok, scale, scale_ref, dispatch, group);
        for (int k = tid; k < kMiscInts; k += 1024) misc[k] = 0;
    } else {
        s_ref = *s_ref_p;
    }
    for (int b = tid; b <= n_buckets; b += 1024) s_start[b] = 0;
    __syncthreads();
    for (int n = tid; n < n_vis; n += 1024) {
        const double2 p = uv[n];
        const int b = bucket_coord(p.y, s_ref, g.inv_du, g.N, nb) * nb + bucket_coord(p.x, s_ref, g.inv_du, g.N, nb);
        s_bkt[n] = (unsigned short)b;
        atomicAdd(&s_start[b], 1);
    }
    __syncthreads();
    // exclusive scan of up to 4096 counts: 4 per thread, warp scan, scan of the warp sums
    {
        const int i0 = tid * 4;
        int v[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) v[k] = (i0 + k < n_buckets) ? s_start[i0 + k] : 0;
        const int tsum = v[0] + v[1] + v[2] + v[3];
        int inc = tsum;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += t;
        }
        if (lane == 31) s_warp[wid] = inc;
        __syncthreads();
        if (wid == 0) {
            int ws = s_warp[lane];
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int t = __shfl_up_sync(0xffffffffu, ws, o);
                if (lane >= o) ws += t;
            }
            s_warp[lane] = ws;
        }
        __syncthreads();
        int excl = (wid > 0 ? s_warp[wid - 1] : 0) + inc - tsum;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            if (i0 + k < n_buckets) { s_start[i0 + k] = excl; s_cursor[i0 + k] = excl; bucket_start[i0 + k] = excl; }
            excl += v[k];
        }
        if (tid == 0) { s_start[n_buckets] = n_vis; bucket_start[n_buckets] = n_vis; }
    }
    __syncthreads();
    for (int n = tid; n < n_vis; n += 1024) s_tmp[atomicAdd(&s_cursor[s_bkt[n]], 1)] = (unsigned short)n;
    __syncthreads();
    // ascending row order inside every bucket: rank = number of smaller row ids of the same bucket
    for (int i = tid; i < n_vis; i += 1024) {
        const int row = s_tmp[i], b = s_bkt[row];
        const int k0 = s_start[b], k1 = s_start[b + 1];
        int rank = 0;
        for (int j = k0; j < k1; ++j) rank += s_tmp[j] < row;
        const double2 p = uv[row];
        perm[k0 + rank] = row;
        uv_sorted[k0 + rank] = p;
        row_sorted[k0 + rank] = make_double4(p.x, p.y, (double)row, 0.0);
    }
    // tile weights (rows whose bucket lies under the tile) and the heaviest-first order (ties by tile index)
    const int per = kTile / kBucketCells;
    for (int t = tid; t < n_tiles; t += 1024) {
        const int ty = t / nt, tx = t - ty * nt;
        int w = 0;
        for (int dy = 0; dy < per; ++dy) {
            const int by = ty * per + dy;
            if (by >= nb) break;
            const int b0 = by * nb + tx * per, b1 = by * nb + min(nb, tx * per + per);
            if (b0 < b1) w += s_start[b1] - s_start[b0];
        }
        s_tw[t] = w;
        tile_weight[t] = w;
    }
    __syncthreads();
    for (int t = tid; t < n_tiles; t += 1024) {
        const int w = s_tw[t];
        int rank = 0;
        for (int u = 0; u < n_tiles; ++u) rank += (s_tw[u] > w) || (s_tw[u] == w && u < t);
        tile_order[rank] = t;
    }
}

bool binning_is_small(const Plan* p, long long n_vis) {
    const int nb = (p->geom.N + kBucketCells - 1) / kBucketCells, nt = (p->geom.N + kTile - 1) / kTile;
    return n_vis > 0 && n_vis <= kSmallRows && nb * nb <= kSmallBuckets && nt * nt <= kSmallTiles;
}

// a1 + a3 of a small call (binning_is_small) in one launch; writes what launch_scale + launch_binning write
bool launch_small_prepass(Plan* p, const double* uv, const double* freqs, long long n_vis, int n_chan, cudaStream_t st) {
    Workspace& ws = p->ws;
    const int nb = (p->geom.N + kBucketCells - 1) / kBucketCells, nt = (p->geom.N + kTile - 1) / kTile;
    bin_small_kernel<<<1, 1024, 0, st>>>(p->geom, (const double2*)uv, nullptr, (int)n_vis, nb, nt, ws.d_bucket_count, ws.d_perm,
                                         ws.d_uv_sorted, (double4*)ws.d_row_sorted, ws.d_tile_weight, ws.d_tile_order, freqs, n_chan,
                                         (chan_supported(p, n_chan) || chanws_supported(p, n_chan)) ? 1 : 0, ws.d_scale, ws.d_scale_ref,
                                         ws.d_dispatch, (double4*)ws.d_group, ws.d_misc);
    p->last_launches += 1;
    p->pdl_next = true;
    return cuda_ok(cudaGetLastError(), "bin_small_kernel (fused pre-pass)");
}

// The two memsets of the multi-kernel binning path, for callers that enqueue them BEFORE scale_kernel: bin_count_kernel
// can then be launched as scale_kernel's programmatic dependent (launch_binning with cleared = true).
bool launch_binning_clear(Plan* p, cudaStream_t st) {
    Workspace& ws = p->ws;
    const int nb = (p->geom.N + kBucketCells - 1) / kBucketCells;
    if (!cuda_ok(cudaMemsetAsync(ws.d_misc, 0, (size_t)kMiscInts * sizeof(int), st), "memset misc")) return false;
    if (!cuda_ok(cudaMemsetAsync(ws.d_bucket_count, 0, ((size_t)nb * nb + 1) * sizeof(int), st), "memset buckets")) return false;
    p->last_launches += 2;
    return true;
}

bool launch_binning(Plan* p, const double* uv, long long n_vis, int /*n_chan*/, cudaStream_t st, bool cleared) {
    Workspace& ws = p->ws;
    const int nb = (p->geom.N + kBucketCells - 1) / kBucketCells;
    const int n_buckets = nb * nb;
    const int nt = (p->geom.N + kTile - 1) / kTile;
    if (!cleared && !cuda_ok(cudaMemsetAsync(ws.d_misc, 0, (size_t)kMiscInts * sizeof(int), st), "memset misc")) return false;
    if (!cleared && n_vis <= kSmallRows && n_buckets <= kSmallBuckets && nt * nt <= kSmallTiles) {
        bin_small_kernel<<<1, 1024, 0, st>>>(p->geom, (const double2*)uv, ws.d_scale_ref, (int)n_vis, nb, nt, ws.d_bucket_count,
                                             ws.d_perm, ws.d_uv_sorted, (double4*)ws.d_row_sorted, ws.d_tile_weight, ws.d_tile_order,
                                             nullptr, 0, 0, nullptr, nullptr, nullptr, nullptr, nullptr);
        p->last_launches += 2;
        return cuda_ok(cudaGetLastError(), "bin_small_kernel");
    }
    if (!cleared && !cuda_ok(cudaMemsetAsync(ws.d_bucket_count, 0, ((size_t)n_buckets + 1) * sizeof(int), st), "memset buckets"))
        return false;
    int blocks = (int)((n_vis + 255) / 256);
    if (blocks > p->sm_count * 8) blocks = p->sm_count * 8;
    // every kernel is launched as a programmatic dependent of the one before it: it becomes resident while its predecessor
    // drains and waits (pdl_wait) for the predecessor's completion before its first read.  bin_count_kernel joins the chain
    // behind scale_kernel when the memsets were enqueued before that kernel (cleared), else it follows the memsets plainly.
    cudaError_t e = cudaSuccess;
    if (cleared)
        e = launch_dependent(bin_count_kernel, dim3(blocks), dim3(256), 0, st, p->geom, (const double2*)uv, (const double*)ws.d_scale_ref,
                             (int)n_vis, nb, ws.d_bucket_count);
    else
        bin_count_kernel<<<blocks, 256, 0, st>>>(p->geom, (const double2*)uv, ws.d_scale_ref, (int)n_vis, nb, ws.d_bucket_count);
    if (e == cudaSuccess) e = launch_dependent(bin_scan_kernel, dim3((n_buckets + kScanPerBlock - 1) / kScanPerBlock), dim3(1024), 0, st,
                                     ws.d_bucket_count, n_buckets, ws.d_bucket_cursor, ws.d_misc + kMiscScanState);
    if (e == cudaSuccess)
        e = launch_dependent(bin_scatter_kernel, dim3(blocks), dim3(256), 0, st, p->geom, (const double2*)uv, (const double*)ws.d_scale_ref,
                             (int)n_vis, nb, ws.d_bucket_cursor, ws.d_perm_tmp);
    {
        long long oblocks = ((long long)n_buckets * 32 + 255) / 256;
        if (oblocks > p->sm_count * 16) oblocks = p->sm_count * 16;
        if (e == cudaSuccess)
            e = launch_dependent(bin_order_kernel, dim3((unsigned)oblocks), dim3(256), 0, st, (const double2*)uv, (const int*)ws.d_bucket_count,
                                 n_buckets, (const int*)ws.d_perm_tmp, ws.d_perm, ws.d_uv_sorted, (double4*)ws.d_row_sorted,
                                 ws.d_misc + kMiscBigList);
        if (n_vis > kOrderWarpMax) {                           // else no bucket can be big
            if (e == cudaSuccess)
                e = launch_dependent(bin_order_large_kernel, dim3(p->sm_count), dim3(1024), 0, st, (const double2*)uv,
                                     (const int*)ws.d_bucket_count, ws.d_perm_tmp, ws.d_perm, ws.d_uv_sorted, (double4*)ws.d_row_sorted,
                                     (const int*)(ws.d_misc + kMiscBigList));
            p->last_launches += 1;
        }
    }
    int* hist = ws.d_misc + 16;
    int tblocks = (nt * nt + 255) / 256;
    if (tblocks > p->sm_count * 8) tblocks = p->sm_count * 8;
    if (e == cudaSuccess)
        e = launch_dependent(tile_weight_kernel, dim3(tblocks), dim3(256), 0, st, (const int*)ws.d_bucket_count, nb, nt, ws.d_tile_weight, hist);
    if (e == cudaSuccess) e = launch_dependent(tile_order_scan_kernel, dim3(1), dim3(kWeightBins), 0, st, hist);
    if (e == cudaSuccess)
        e = launch_dependent(tile_order_scatter_kernel, dim3(tblocks), dim3(256), 0, st, (const int*)ws.d_tile_weight, nt * nt, hist,
                             ws.d_tile_order);
    if (!cuda_ok(e, "binning kernels (dependent launches)")) return false;
    p->pdl_next = true;                                        // a gridder that comes next may join the chain
    p->last_launches += cleared ? 7 : 9;
    return cuda_ok(cudaGetLastError(), "binning kernels");
}

}  // namespace mwa
