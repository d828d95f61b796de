// k_gather.cu - K3c, the product gridder: tile-owned, register-resident accumulation (a2 + a4 + a5 fused).
//
// One WARP owns one 16x16-cell tile of one channel (all 4 polarisations) from its first tap to its single
// write-out, so there are no atomics on grid data anywhere and every grid cell is written exactly once,
// zeros included (R10; SURVEY.md section 7 hard part 2).  Inside the warp every lane owns a 4x2 block
// of cells: 8 cells x 4 pol x (re, im) = 64 fp32 accumulators in registers.  PAPER.md:49 calls this the
// "gather" form ("a thread collects the values for a particular memory location"); what is new here is
// how a lane finds its values without scanning everything:
//
//   phase A (lane = candidate row): walk the buckets of k_bin.cu that can reach the tile at this channel's
//            scale - in a fixed scattered order, groups of 8 sorted rows at a time, so that a buffer of 128 hits is a
//            spatially mixed sample and the per-lane lists of phase B are balanced - run the exact index function
//            (index.cuh) on each candidate, keep the rows whose WxW stamp overlaps the tile; per hit store the table
//            offsets and a 32-bit mask of the lanes (4x2 blocks) the stamp overlaps, and request its visibilities and
//            weight with cp.async straight into the buffer (they land while the scan goes on).
//   transpose: a 32x32 bit-matrix transpose by warp shuffles turns "blocks per hit" into "hits per block".
//   phase B (lane = block owner): each lane walks ITS OWN hit list, branch-free: a lane whose list is exhausted takes
//            a null hit (zero visibility, zero weight), so the warp runs one instruction stream with two operand sets in
//            flight.  Per visit a lane reads V (2 x LDS.128 from the two half planes), geo + weight (LDS.64), 4 u-taps
//            (LDS.128) and 2 v-taps (LDS.64) from zero-padded, pre-shifted copies of the kernel table, and issues 10 FMUL
//            and 32 packed fma.rn.f32x2.
//   write-out: 16 x STG.128 per lane, streaming (evict-first) so the grid does not push vis lines out of L2; with
//            accumulate-into a read-modify-write of the warp's own cells; with multi-frequency synthesis (all channels
//            onto one grid) a red.global.add.v4.f32 per 16 B.
//
// Work items (tile, channel) are taken from a global counter up to 8 at a time, channel fastest, tiles heaviest first.
// Calls with few items per warp run the instantiation gather_kernel<true>: the items of the heavy tiles come first and
// are gridded by the four warps of a CTA together ("heavy items" in the kernel).  Behind a pre-pass chain of programmatic
// dependent launches (plan.h) the kernel builds its table copies before griddepcontrol.wait (GatherParams::pdl).
// profiles/r02_gather_c5.md: C5 in 23.0 ms (round 1: 36.4 ms); bound by the shared-memory pipe (the LDS of phase B are
// lane-scattered by construction).
#include <cstdint>

#include "plan.h"

namespace mwa {

constexpr int kWarpsPerCta = 4;
constexpr int kCap = 128;                 // hits buffered per warp before they are consumed
constexpr int kBlocksX = 4, kBlocksY = 8; // lane -> block (bx = lane & 3, by = lane >> 2); block = 4 x 2 cells

struct GatherParams {
    GridGeom g;
    const double* scale;        // [n_chan]
    const double* scale_ref;    // [1]
    const int* bucket_start;    // [nb*nb + 1]
    const int* perm;            // [n_vis]
    const double2* uv_sorted;   // [n_vis]
    const int* tile_order;      // [nt*nt]
    int* counter;               // work counter
    const int* dispatch;        // AUTO: run only if *dispatch == 0 (see scale_kernel); null = always
    const float4* vis;          // [n_vis][n_chan][2] float4
    const float* weights;       // [n_vis][n_chan] or null
    const float* table;         // [(O+1)][W]
    float* grid;                // [n_chan][4][N][N][2]
    int n_chan, nb, nt;
    int rlu, rlv;               // padded row lengths of the shifted table copies
    long long n_items;
    int accumulate;             // 1: grid += (f3 accumulate-into), 0: grid = (R10)
    int mfs;                    // 1: all channels add into ONE grid [4][N][N] (f3 multi-frequency synthesis): the write-out of a
                                //    (tile, channel) item is a reduction (red.global.add.v4.f32) into the zero-filled shared grid
    int chunk;                  // consecutive work items per claim (1..8; amortises the round trip of the work counter)
    const int* heavy_tiles;     // null, or [1]: the first *heavy_tiles entries of tile_order are heavy tiles (weight >= kHeavyTileWeight):
                                //    each of their items is gridded by the FOUR warps of a CTA together (see "heavy items" below)
    int* heavy_counter;         // work counter of the heavy items
    int v8;                     // 1: N % 4 == 0 and grid 32-byte aligned: the write-out uses 256-bit stores (one full sector per lane)
    int pdl;                    // 1: launched with programmatic stream serialisation behind the fused pre-pass of a small call
                                //    (bin_small_kernel): the table copies are built while the pre-pass still runs, and
                                //    griddepcontrol.wait comes before the first read of anything the pre-pass writes
};

typedef unsigned long long u64;

__device__ __forceinline__ u64 pack2(float a, float b) {
    u64 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b));
    return r;
}
__device__ __forceinline__ void unpack2(u64 v, float& a, float& b) {
    asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v));
}
__device__ __forceinline__ void ffma2(u64& d, u64 a, u64 b) {        // d = a * b + d, two fp32 lanes
    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(d) : "l"(a), "l"(b));
}
__device__ __forceinline__ void st_stream_v4(float* p, float a, float b, float c, float d) {
    asm volatile("st.global.cs.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
}

// 32x32 bit-matrix transpose across the warp: in = row `lane`, out bit h = bit `lane` of lane h's input.
__device__ __forceinline__ unsigned transpose32(unsigned x, int lane) {
#pragma unroll
    for (int s = 0; s < 5; ++s) {
        const int j = 16 >> s;
        const unsigned m = s == 0 ? 0x0000FFFFu : s == 1 ? 0x00FF00FFu : s == 2 ? 0x0F0F0F0Fu : s == 3 ? 0x33333333u : 0x55555555u;
        const unsigned y = __shfl_xor_sync(0xffffffffu, x, j);
        x = (lane & j) ? ((x & ~m) | ((y >> j) & m)) : ((x & m) | ((y << j) & ~m));
    }
    return x;
}

struct WarpSmem {
    float4 z[2][kCap + 1];  // V by halves: [0] {XX.re, XX.im, XY.re, XY.im}, [1] {YX.re, YX.im, YY.re, YY.im} (cp.async from
                            // phase A); 16 B per hit and half, so the lane-private LDS.128 of phase B spread over all banks
    uint2 gw[kCap + 1];     // x: (byte offset into u copies + bias) | (byte offset into v copies + bias) << 16; y: weight
                            // (cp.async); one LDS.64 per visit
    unsigned mask[kCap];    // lanes (blocks) the stamp overlaps
};

constexpr int kBiasU = 16, kBiasV = 16;   // floats; keep the stored offsets non-negative

// kHeavy: the instantiation with the CTA-cooperative heavy items in front of the per-warp items (launched only for calls
// with few items per warp; 3 CTAs per SM so that the second code path does not spill)
template <bool kHeavy>
__global__ void __launch_bounds__(kWarpsPerCta * 32, kHeavy ? 3 : 4)
gather_kernel(const GatherParams P) {
    if (!P.pdl && P.dispatch != nullptr && *P.dispatch != 0) return;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const GridGeom g = P.g;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    // ---- shifted, zero-padded table copies (built once per CTA)
    //   tu[s][r][q] = Tp_u[r][q + s], Tp_u[r][3 + t] = T[r][t]      s = 0..3, q = 0..rlu-1
    //   tv[s][r][q] = Tp_v[r][q + s], Tp_v[r][1 + t] = T[r][t]      s = 0..1, q = 0..rlv-1
    float* tu = reinterpret_cast<float*>(smem_raw);
    const int n_tu = 4 * (g.O + 1) * P.rlu;
    const int n_tv = 2 * (g.O + 1) * P.rlv;
    float* tv = tu + n_tu;
    WarpSmem* wsm = reinterpret_cast<WarpSmem*>(smem_raw + (((size_t)(n_tu + n_tv) * 4 + 15) & ~size_t(15))) + warp;
    for (int k = threadIdx.x; k < n_tu; k += blockDim.x) {
        const int q = k % P.rlu, r = (k / P.rlu) % (g.O + 1), s = k / (P.rlu * (g.O + 1));
        const int t = q + s - 3;
        tu[k] = (t >= 0 && t < g.W) ? P.table[r * g.W + t] : 0.0f;
    }
    for (int k = threadIdx.x; k < n_tv; k += blockDim.x) {
        const int q = k % P.rlv, r = (k / P.rlv) % (g.O + 1), s = k / (P.rlv * (g.O + 1));
        const int t = q + s - 1;
        tv[k] = (t >= 0 && t < g.W) ? P.table[r * g.W + t] : 0.0f;
    }
    __syncthreads();
    if (P.pdl) {                                             // the pre-pass has completed and its writes are visible from here on
        asm volatile("griddepcontrol.wait;" ::: "memory");
        if (P.dispatch != nullptr && *P.dispatch != 0) return;
    }

    const int bx = lane & 3, by = lane >> 2;
    const unsigned tu_s = (unsigned)__cvta_generic_to_shared(tu);
    const unsigned tv_s = (unsigned)__cvta_generic_to_shared(tv);
    const unsigned z_s = (unsigned)__cvta_generic_to_shared(&wsm->z[0][0]);
    const unsigned gw_s = (unsigned)__cvta_generic_to_shared(&wsm->gw[0]);
    constexpr unsigned kZHalf = 16u * (kCap + 1);
    const bool has_w = P.weights != nullptr;
    // lane constants of the table addresses: offset (floats) = stored - bias + 4*bx  (u), + 2*by (v)
    const unsigned cu = tu_s + (unsigned)((4 * bx - kBiasU) * 4);
    const unsigned cv = tv_s + (unsigned)((2 * by - kBiasV) * 4);
    if (lane == 0) {                                     // the null hit of phase B
        wsm->z[0][kCap] = make_float4(0.f, 0.f, 0.f, 0.f);
        wsm->z[1][kCap] = make_float4(0.f, 0.f, 0.f, 0.f);
        wsm->gw[kCap] = make_uint2((unsigned)(kBiasU * 4) | ((unsigned)(kBiasV * 4) << 16), 0u);
    }
    __syncwarp();
    const double s_ref = *P.scale_ref;
    const size_t plane = (size_t)g.N * g.N;
    const unsigned lt_mask = (1u << lane) - 1u;

    // ---- heavy items.  With few work items per warp (one channel, a large grid: C3) the call lasts as long as its
    // heaviest tile takes ONE warp - thousands of hits against a mean of a hundred.  The items of the heavy tiles (the
    // head of tile_order) are therefore taken first, one per CTA: warp k walks every fourth round of 32 candidates
    // (slice k), the four register tiles are added in shared memory in the fixed order 0 + 1 + 2 + 3 (deterministic),
    // and warp 0 writes the tile.  A CTA that finds no heavy item left goes on to the per-warp items below.
    __shared__ long long s_heavy_item;
    __shared__ int s_any_hit[kWarpsPerCta];
    u64* red = reinterpret_cast<u64*>(wsm - warp + kWarpsPerCta);      // [3][32][32] u64 behind the WarpSmem array (heavy only)
    bool heavy = kHeavy;                                                 // CTA-uniform; constant false in the plain instantiation
    const long long n_heavy = heavy ? (long long)(*P.heavy_tiles) * P.n_chan : 0;   // normal items start here
    if (kHeavy && blockIdx.x == 0 && threadIdx.x == 0)                   // diagnostics: mwa_grid_plan_last_stats()[31]
        *reinterpret_cast<long long*>(P.heavy_counter - kMiscHeavyCounter + kMiscHeavyStat) = n_heavy;

    long long base = 0;
    int sub = 0;
    long long next_base = 0;
    if (!heavy) {
        if (lane == 0) base = (long long)atomicAdd(P.counter, P.chunk);
        base = __shfl_sync(0xffffffffu, base, 0);
    }

    while (true) {
        long long item;
        if (heavy) {
            __syncthreads();                                             // s_heavy_item and red[] of the item before are free
            if (threadIdx.x == 0) s_heavy_item = (long long)atomicAdd(P.heavy_counter, 1);
            __syncthreads();
            item = s_heavy_item;
            if (item >= n_heavy) {                                       // on to the per-warp items
                heavy = false;
                if (lane == 0) base = (long long)atomicAdd(P.counter, P.chunk);
                base = __shfl_sync(0xffffffffu, base, 0);
                sub = 0;
                continue;
            }
        } else {
            item = n_heavy + base + sub;
            if (item >= P.n_items) break;
            if (sub == 0 && lane == 0) next_base = (long long)atomicAdd(P.counter, P.chunk);   // used P.chunk items from now
        }
        const int nsl = heavy ? kWarpsPerCta : 1, slice = heavy ? warp : 0;
        const int trank = (int)(item / P.n_chan);
        const int c = (int)(item - (long long)trank * P.n_chan);
        const int tile = P.tile_order[trank];
        const int ty = tile / P.nt, tx = tile - ty * P.nt;
        const int X0 = tx * kTile, Y0 = ty * kTile;
        const double sc = P.scale[c];

        // ---- candidate buckets: back-project [X0 - h - 1, X0 + 15 + h + 1] (cells from the centre) to s_ref
        int bx0 = 0, bx1 = P.nb - 1, by0 = 0, by1 = P.nb - 1;
        {
            const double rho = sc / s_ref;                       // <= 1 for positive frequencies
            if (rho > 1e-3 && rho <= 1.0 + 1e-9) {
                const double half = (double)(g.N / 2), pad = (double)g.h + 1.25, inv = 1.0 / rho;
                const double lox = ((double)X0 - pad - half) * inv + half, hix = ((double)(X0 + kTile - 1) + pad - half) * inv + half;
                const double loy = ((double)Y0 - pad - half) * inv + half, hiy = ((double)(Y0 + kTile - 1) + pad - half) * inv + half;
                const double ib = 1.0 / kBucketCells, top = (double)(P.nb - 1);
                bx0 = (int)fmin(fmax(floor(lox * ib), 0.0), top);
                bx1 = (int)fmin(fmax(floor(hix * ib), 0.0), top);
                by0 = (int)fmin(fmax(floor(loy * ib), 0.0), top);
                by1 = (int)fmin(fmax(floor(hiy * ib), 0.0), top);
            }
        }

        u64 acc[2][4][4];   // [row i][col j][pol] = (re, im)
#pragma unroll
        for (int i = 0; i < 2; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j)
#pragma unroll
                for (int p = 0; p < 4; ++p) acc[i][j][p] = 0ull;

        int n_buf = 0;
        bool any_hit = false;                                              // MFS: an item without hits has nothing to add

        // consume the buffered hits: loads of w*V, transpose, per-lane walk
        auto consume = [&](int n) {
            // the visibilities and weights of the buffered hits were requested with cp.async when the hits were found
            asm volatile("cp.async.wait_all;" ::: "memory");
            __syncwarp();
            unsigned mw[kCap / 32];
#pragma unroll
            for (int b = 0; b < kCap / 32; ++b) {
                const int hidx = b * 32 + lane;
                const unsigned m = (b * 32 < n) ? ((hidx < n) ? wsm->mask[hidx] : 0u) : 0u;
                mw[b] = (b * 32 < n) ? transpose32(m, lane) : 0u;
            }
            __syncwarp();
            // ---- phase B: every lane walks its own hit list, branch-free.  A lane whose list is exhausted (or whose current
            // mask word is) takes the null hit - slot kCap: zero visibilities, zero weight, an in-range table offset - so the
            // whole warp runs the same instruction stream for `steps` rounds, the longest list plus its empty words.  The
            // loads of a visit are issued under the FMAs of the visit before it (two operand sets, as K6's consumers).
            unsigned m = mw[0], q1 = mw[1], q2 = mw[2], q3 = mw[3];
            int wb = 0;
            int mine = __popc(m) + __popc(q1) + __popc(q2) + __popc(q3);
            mine += (m == 0u ? 1 : 0) + (q1 == 0u ? 1 : 0) + (q2 == 0u ? 1 : 0);      // a step that only moves on to the next word
            const int steps = __reduce_max_sync(0xffffffffu, mine);
            auto next_hit = [&]() -> unsigned {
                const bool refill = m == 0u;
                m = refill ? q1 : m; q1 = refill ? q2 : q1; q2 = refill ? q3 : q2; q3 = refill ? 0u : q3;
                wb += refill ? 32 : 0;
                const unsigned bit = (unsigned)(__ffs(m) - 1);
                const unsigned hidx = m != 0u ? (unsigned)wb + bit : (unsigned)kCap;
                m &= m - 1u;
                return hidx;
            };
#define K3_GW(h, G, WT) asm volatile("ld.shared.v2.b32 {%0, %1}, [%2];" : "=r"(G), "=r"(WT) : "r"(gw_s + 8u * (h)));
#define K3_LOAD(h, g, Z0, Z1, Z2, Z3, U0, U1, U2, U3, V0, V1)                                                              \
    asm volatile("ld.shared.v2.b64 {%0, %1}, [%2];" : "=l"(Z0), "=l"(Z1) : "r"(z_s + 16u * (h)));                           \
    asm volatile("ld.shared.v2.b64 {%0, %1}, [%2];" : "=l"(Z2), "=l"(Z3) : "r"(z_s + kZHalf + 16u * (h)));                  \
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(U0), "=f"(U1), "=f"(U2), "=f"(U3) : "r"(cu + ((g) & 0xffffu))); \
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(V0), "=f"(V1) : "r"(cv + ((g) >> 16)));
#define K3_FMA(Z0, Z1, Z2, Z3, U0, U1, U2, U3, V0, V1, WT)                                                                 \
    {                                                                                                                      \
        const float kvw[2] = {V0 * __uint_as_float(WT), V1 * __uint_as_float(WT)};                                                                         \
        const float kuu[4] = {U0, U1, U2, U3};                                                                             \
        _Pragma("unroll") for (int i = 0; i < 2; ++i) _Pragma("unroll") for (int j = 0; j < 4; ++j) {                       \
            const float kq = kvw[i] * kuu[j];                                                                              \
            const u64 kk = pack2(kq, kq);                                                                                  \
            ffma2(acc[i][j][0], kk, Z0);                                                                                   \
            ffma2(acc[i][j][1], kk, Z1);                                                                                   \
            ffma2(acc[i][j][2], kk, Z2);                                                                                   \
            ffma2(acc[i][j][3], kk, Z3);                                                                                   \
        }                                                                                                                  \
    }
            if (steps > 0) {
                u64 az0, az1, az2, az3, bz0, bz1, bz2, bz3;
                float au0, au1, au2, au3, av0, av1, bu0, bu1, bu2, bu3, bv0, bv1;
                unsigned aw, bw;                                           // weights (bits) of the visits in flight
                const unsigned h0 = next_hit();
                unsigned h1 = next_hit(), h2 = next_hit();
                unsigned g1, g2, w2;
                {
                    unsigned g0;
                    K3_GW(h0, g0, aw)
                    K3_GW(h1, g1, bw)
                    K3_LOAD(h0, g0, az0, az1, az2, az3, au0, au1, au2, au3, av0, av1)
                }
#pragma unroll 1
                for (int v = 0; v < steps; v += 2) {
                    K3_LOAD(h1, g1, bz0, bz1, bz2, bz3, bu0, bu1, bu2, bu3, bv0, bv1)
                    K3_GW(h2, g2, w2)
                    const unsigned h3 = next_hit();
                    K3_FMA(az0, az1, az2, az3, au0, au1, au2, au3, av0, av1, aw)
                    if (v + 1 >= steps) break;
                    aw = w2;
                    K3_LOAD(h2, g2, az0, az1, az2, az3, au0, au1, au2, au3, av0, av1)
                    const unsigned wb_cur = bw;
                    K3_GW(h3, g1, bw)
                    const unsigned h4 = next_hit();
                    K3_FMA(bz0, bz1, bz2, bz3, bu0, bu1, bu2, bu3, bv0, bv1, wb_cur)
                    h1 = h3;
                    h2 = h4;
                }
            }
#undef K3_GW
#undef K3_LOAD
#undef K3_FMA
            __syncwarp();
        };

        // ---- phase A, pass 1: lane = candidate.  The candidates of the window (the sorted rows of its bucket rows, `total`
        // of them) are visited in a fixed scattered order, position j -> candidate (j * S) mod total with S ~ 0.618 total
        // coprime to total, not bucket after bucket: the hits of one bucket have nearly the same stamp origin and fall on the
        // same few 4 x 2 blocks, so a buffer filled in sorted order keeps a few lanes busy in phase B while the others
        // idle.  A pure function of the sorted rows: the result stays bit-identical from run to run.
        for (int rg = by0; rg <= by1; rg += 32) {
            int k0 = 0, len = 0;
            if (rg + lane <= by1) {                                          // lane = bucket row rg + lane
                k0 = __ldg(P.bucket_start + (rg + lane) * P.nb + bx0);
                len = __ldg(P.bucket_start + (rg + lane) * P.nb + bx1 + 1) - k0;
            }
            int incl = len;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int t = __shfl_up_sync(0xffffffffu, incl, o);
                if (lane >= o) incl += t;
            }
            const int total = __shfl_sync(0xffffffffu, incl, 31);
            const int excl = incl - len;
            if (total == 0) continue;
            // groups of 8 consecutive candidates (one 128 B line of uv records, one sector of row ids) are the unit that is
            // scattered: group position gj -> group (gj * S) mod ng
            const int ng = (total + 7) >> 3;
            int S = 1;
            if (ng >= 8) {
                S = (int)(((long long)ng * 618) / 1000) | 1;
                for (;; S += 2) {
                    int ga = ng, gb = S;
                    while (gb) { const int t = ga % gb; ga = gb; gb = t; }
                    if (ga == 1) break;
                }
            }
            const int gstep = (int)(((long long)(4 * nsl) * S) % ng);          // a round of 32 candidates is 4 groups; every nsl-th round
            int gp = (int)(((long long)((lane >> 3) + 4 * slice) * S) % ng);   // the lane's current group
            int f = gp * 8 + (lane & 7);
            auto locate = [&](int cb, int& row, double2& p) {
                int lo = 0;                                                  // smallest bucket row with incl > f
#pragma unroll
                for (int st = 16; st > 0; st >>= 1) {
                    const int t = __shfl_sync(0xffffffffu, incl, lo + st - 1);
                    if (t <= f) lo += st;
                }
                lo = min(lo, 31);
                const int k = __shfl_sync(0xffffffffu, k0, lo) + (f - __shfl_sync(0xffffffffu, excl, lo));
                p = make_double2(0.0, 0.0);
                row = -1;                                                    // -1: no candidate at this position
                if ((cb >> 3) + (lane >> 3) < ng && f < total) { p = __ldg(P.uv_sorted + k); row = __ldg(P.perm + k); }   // positions >= ng would wrap around
                gp += gstep;
                if (gp >= ng) gp -= ng;
                f = gp * 8 + (lane & 7);
            };
            int row_nx;
            double2 p_nx;
            locate(32 * slice, row_nx, p_nx);
            for (int cb = 32 * slice; cb < ng * 8; cb += 32 * nsl) {
                const int row = row_nx;
                const bool in_range = row >= 0;
                const double2 p = p_nx;
                if (cb + 32 * nsl < ng * 8) locate(cb + 32 * nsl, row_nx, p_nx);
                bool hit = false;
                unsigned geo = 0, mask = 0;
                if (in_range) {
                    SampleIndex s;
                    if (sample_index(p.x, p.y, sc, g, s)) {
                        const int ou = s.iu - g.h - X0, ov = s.iv - g.h - Y0;     // stamp origin relative to the tile
                        if (ou > -g.W && ou < kTile && ov > -g.W && ov < kTile) {
                            hit = true;
                            const int su = (3 - ou) & 3, sv = (1 - ov) & 1;
                            const int offu = (su * (g.O + 1) + s.ru) * P.rlu + (3 - ou - su) + kBiasU;
                            const int offv = (sv * (g.O + 1) + s.rv) * P.rlv + (1 - ov - sv) + kBiasV;
                            geo = (unsigned)(offu * 4) | ((unsigned)(offv * 4) << 16);
                            const int bxl = max(0, ou >> 2), bxh = min(kBlocksX - 1, (ou + g.W - 1) >> 2);
                            const int byl = max(0, ov >> 1), byh = min(kBlocksY - 1, (ov + g.W - 1) >> 1);
                            const unsigned m4 = (2u << bxh) - (1u << bxl);
                            const unsigned rows = 0x11111111u & (0xFFFFFFFFu >> (28 - 4 * byh)) & (0xFFFFFFFFu << (4 * byl));
                            mask = rows * m4;
                        }
                    }
                }
                const unsigned ball = __ballot_sync(0xffffffffu, hit);
                const int cnt = __popc(ball);
                if (cnt == 0) continue;
                any_hit = true;
                if (n_buf + cnt > kCap) { consume(n_buf); n_buf = 0; }
                if (hit) {
                    const int slot = n_buf + __popc(ball & lt_mask);
                    wsm->gw[slot].x = geo;
                    wsm->mask[slot] = mask;
                    // the sample's 32 B of visibilities and its weight go straight to the buffer, asynchronously: they land
                    // while the scan goes on
                    const size_t sidx = (size_t)row * P.n_chan + c;
                    const float4* src = P.vis + 2 * sidx;
#ifdef K3_NO_L2_PREFETCH
                    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(z_s + 16u * slot), "l"(src) : "memory");
                    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(z_s + kZHalf + 16u * slot), "l"(src + 1) : "memory");
                    if (has_w) asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(gw_s + 8u * slot + 4u), "l"(P.weights + sidx) : "memory");
#else
                    // .L2::128B: a miss brings the whole 128 B line into L2 - the same sample's next 3 channels (visibilities)
                    // or 31 channels (weights), which the items claimed with this one ask for within microseconds
                    asm volatile("cp.async.cg.shared.global.L2::128B [%0], [%1], 16;" ::"r"(z_s + 16u * slot), "l"(src) : "memory");
                    asm volatile("cp.async.cg.shared.global.L2::128B [%0], [%1], 16;" ::"r"(z_s + kZHalf + 16u * slot), "l"(src + 1) : "memory");
                    if (has_w) asm volatile("cp.async.ca.shared.global.L2::128B [%0], [%1], 4;" ::"r"(gw_s + 8u * slot + 4u), "l"(P.weights + sidx) : "memory");
#endif
                    else wsm->gw[slot].y = __float_as_uint(1.0f);
                }
                n_buf += cnt;
            }
        }
        if (n_buf > 0) consume(n_buf);

        if (heavy) {                                                       // add the four warps' register tiles, in warp order
            if (warp > 0) {
#pragma unroll
                for (int i = 0; i < 2; ++i)
#pragma unroll
                    for (int j = 0; j < 4; ++j)
#pragma unroll
                        for (int q = 0; q < 4; ++q) red[((warp - 1) * 32 + (i * 16 + j * 4 + q)) * 32 + lane] = acc[i][j][q];
            }
            if (lane == 0) s_any_hit[warp] = any_hit ? 1 : 0;
            __syncthreads();
            if (warp > 0) continue;                                        // (the barrier at the head of the loop comes next)
            const u64 ones = pack2(1.0f, 1.0f);
            for (int w = 0; w < kWarpsPerCta - 1; ++w) {
#pragma unroll
                for (int i = 0; i < 2; ++i)
#pragma unroll
                    for (int j = 0; j < 4; ++j)
#pragma unroll
                        for (int q = 0; q < 4; ++q) ffma2(acc[i][j][q], ones, red[(w * 32 + (i * 16 + j * 4 + q)) * 32 + lane]);   // acc += 1 * partial
            }
            any_hit = (s_any_hit[0] | s_any_hit[1] | s_any_hit[2] | s_any_hit[3]) != 0;
        }

        // ---- a5: write the lane's 4x2 block of all 4 planes, once
        if (P.mfs) {
            if (any_hit) {
                const int x = X0 + 4 * bx;
#pragma unroll
                for (int i = 0; i < 2; ++i) {
                    const int y = Y0 + 2 * by + i;
                    if (y < g.N) {
#pragma unroll
                        for (int p = 0; p < 4; ++p) {
                            float* dst = P.grid + ((size_t)p * plane + (size_t)y * g.N + x) * 2;
                            float a0, a1, a2, a3;
                            if (x + 1 < g.N) {
                                unpack2(acc[i][0][p], a0, a1);
                                unpack2(acc[i][1][p], a2, a3);
                                asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(dst), "f"(a0), "f"(a1), "f"(a2), "f"(a3) : "memory");
                            }
                            if (x + 3 < g.N) {
                                unpack2(acc[i][2][p], a0, a1);
                                unpack2(acc[i][3][p], a2, a3);
                                asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(dst + 4), "f"(a0), "f"(a1), "f"(a2), "f"(a3) : "memory");
                            }
                        }
                    }
                }
            }
        } else if (P.v8) {
            // N is a multiple of 4 and the grid 32-byte aligned: a lane's 4 cells of a row are one aligned 32-byte sector,
            // written by ONE 256-bit store (the four lanes of a block row fill a 128-byte line per instruction; two 128-bit
            // stores would write every sector in two halves, two instructions apart)
            const int x = X0 + 4 * bx;
            if (x < g.N) {
#pragma unroll
                for (int i = 0; i < 2; ++i) {
                    const int y = Y0 + 2 * by + i;
                    if (y < g.N) {
#pragma unroll
                        for (int p = 0; p < 4; ++p) {
                            float* dst = P.grid + (((size_t)c * 4 + p) * plane + (size_t)y * g.N + x) * 2;
                            float a0, a1, a2, a3, a4, a5, a6, a7;
                            unpack2(acc[i][0][p], a0, a1);
                            unpack2(acc[i][1][p], a2, a3);
                            unpack2(acc[i][2][p], a4, a5);
                            unpack2(acc[i][3][p], a6, a7);
                            if (P.accumulate) {                         // the warp owns these cells: a plain read-modify-write
                                const float4 o0 = *reinterpret_cast<const float4*>(dst), o1 = *reinterpret_cast<const float4*>(dst + 4);
                                a0 += o0.x; a1 += o0.y; a2 += o0.z; a3 += o0.w;
                                a4 += o1.x; a5 += o1.y; a6 += o1.z; a7 += o1.w;
                            }
                            asm volatile("st.global.cs.v8.f32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"l"(dst), "f"(a0), "f"(a1), "f"(a2),
                                         "f"(a3), "f"(a4), "f"(a5), "f"(a6), "f"(a7) : "memory");
                        }
                    }
                }
            }
        } else {
            const int x = X0 + 4 * bx;
#pragma unroll
            for (int i = 0; i < 2; ++i) {
                const int y = Y0 + 2 * by + i;
                if (y < g.N) {
#pragma unroll
                    for (int p = 0; p < 4; ++p) {
                        float* dst = P.grid + (((size_t)c * 4 + p) * plane + (size_t)y * g.N + x) * 2;
                        float a0, a1, a2, a3;
                        if (x + 1 < g.N) {
                            unpack2(acc[i][0][p], a0, a1);
                            unpack2(acc[i][1][p], a2, a3);
                            if (P.accumulate) {                             // the warp owns these cells: a plain read-modify-write
                                const float4 o = *reinterpret_cast<const float4*>(dst);
                                a0 += o.x; a1 += o.y; a2 += o.z; a3 += o.w;
                            }
                            st_stream_v4(dst, a0, a1, a2, a3);
                        }
                        if (x + 3 < g.N) {
                            unpack2(acc[i][2][p], a0, a1);
                            unpack2(acc[i][3][p], a2, a3);
                            if (P.accumulate) {
                                const float4 o = *reinterpret_cast<const float4*>(dst + 4);
                                a0 += o.x; a1 += o.y; a2 += o.z; a3 += o.w;
                            }
                            st_stream_v4(dst + 4, a0, a1, a2, a3);
                        }
                    }
                }
            }
        }
        if (!heavy && ++sub == P.chunk) { sub = 0; base = __shfl_sync(0xffffffffu, next_base, 0); }
    }
}

bool launch_gather(Plan* p, const float* vis, const float* w, long long n_vis, int n_chan, float* grid,
                   const int* dispatch, cudaStream_t st) {
    GatherParams P;
    P.g = p->geom;
    P.scale = p->ws.d_scale;
    P.scale_ref = p->ws.d_scale_ref;
    P.bucket_start = p->ws.d_bucket_count;
    P.perm = p->ws.d_perm;
    P.uv_sorted = p->ws.d_uv_sorted;
    P.tile_order = p->ws.d_tile_order;
    P.counter = p->ws.d_misc;
    P.dispatch = dispatch;
    P.vis = (const float4*)vis;
    P.weights = w;
    P.table = p->d_table;
    P.grid = grid;
    P.n_chan = n_chan;
    P.accumulate = p->accumulate ? 1 : 0;
    P.mfs = p->mfs ? 1 : 0;
    P.v8 = (p->geom.N % 4 == 0 && (reinterpret_cast<uintptr_t>(grid) & 31) == 0) ? 1 : 0;
    if (p->mfs && !p->accumulate) {                             // the reductions need a zeroed grid
        if (!cuda_ok(cudaMemsetAsync(grid, 0, (size_t)4 * p->geom.N * p->geom.N * 8, st), "memset grid")) return false;
        p->last_launches += 1;
    }
    P.nb = (p->geom.N + kBucketCells - 1) / kBucketCells;
    P.nt = (p->geom.N + kTile - 1) / kTile;
    P.rlu = (p->geom.W + 6 + 3) & ~3;
    P.rlv = (p->geom.W + 2 + 1) & ~1;
    P.n_items = (long long)P.nt * P.nt * n_chan;
    const size_t tbl = ((size_t)(4 * P.rlu + 2 * P.rlv) * (p->geom.O + 1) * 4 + 15) & ~size_t(15);
    // heavy items (see the kernel): only where a single warp's heaviest tile can be the critical path - few items per warp -
    // and not behind the one-CTA pre-pass of small calls (it does not count the heavy tiles)
    const bool use_heavy = !binning_is_small(p, n_vis) && P.n_items < (long long)p->sm_count * 16 * 32;
    P.heavy_tiles = use_heavy ? p->ws.d_misc + kMiscHeavyTiles : nullptr;
    P.heavy_counter = p->ws.d_misc + kMiscHeavyCounter;
    const size_t smem = tbl + sizeof(WarpSmem) * kWarpsPerCta + (use_heavy ? (size_t)(kWarpsPerCta - 1) * 32 * 32 * 8 : 0);
    // a per-device setting: set on every launch (cheap), so a process that uses several GPUs gets it on each
    void (*kern)(const GatherParams) = use_heavy ? gather_kernel<true> : gather_kernel<false>;
    if (!cuda_ok(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 160 * 1024),
                 "gather smem attribute"))
        return false;
    int ctas_per_sm = 0;
    if (!cuda_ok(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&ctas_per_sm, kern, kWarpsPerCta * 32, smem),
                 "gather occupancy"))
        return false;
    if (ctas_per_sm < 1) { set_error("gather kernel does not fit on an SM"); return false; }
    long long want = (P.n_items + kWarpsPerCta - 1) / kWarpsPerCta;
    long long blocks = (long long)p->sm_count * ctas_per_sm;
    if (blocks > want) blocks = want;
    if (blocks < 1) blocks = 1;
    // items per claim: up to 8 while every warp still gets at least ~16 claims (small problems keep 1)
    long long chunk = P.n_items / (blocks * kWarpsPerCta * 16);
    P.chunk = (int)(chunk < 1 ? 1 : chunk > 8 ? 8 : chunk);
    P.pdl = p->pdl_next ? 1 : 0;
    p->pdl_next = false;
    if (P.pdl) {
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3((unsigned)blocks);
        cfg.blockDim = dim3(kWarpsPerCta * 32);
        cfg.dynamicSmemBytes = smem;
        cfg.stream = st;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        p->last_launches += 1;
        return cuda_ok(cudaLaunchKernelEx(&cfg, kern, P), "gather_kernel (dependent launch)");
    }
    kern<<<(unsigned)blocks, kWarpsPerCta * 32, smem, st>>>(P);
    p->last_launches += 1;
    return cuda_ok(cudaGetLastError(), "gather_kernel");
}

}  // namespace mwa
