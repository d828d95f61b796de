// k_chan.cu - K5, the channel-SIMD register gridder (a2 + a4 + a5 fused) for finely channelised data.
//
// The correlator of PAPER.md:19 delivers 768 channels of 40 kHz: neighbouring channels see the same baseline
// at almost the same (u, v) (u_lambda = u_m * nu / c moves by 2.6e-4 of its radius per channel), and every
// channel owns its own grid (BASELINE.json configs[3]).  K5 turns that into SIMD lanes:
//
//   CTA  = one 16 x 4 cell tile x one SUPER-GROUP of 6 x 32 adjacent channels; 8 warps, 2 CTAs per SM
//   warp = one 4x2-cell block of the tile
//   lane = one channel of the current 32-channel group; the lane keeps 8 cells x 4 pol x (re, im) = 64 fp32
//          accumulators of ITS channel's grid in registers.
//
// All 32 lanes of a warp therefore walk (almost) the same list of baseline rows - the walk is balanced by
// construction, where K3c (k_gather.cu: lane = block, same channel) leaves 23 of 32 lanes idle on Poisson
// noise (profiles/r01_gather_v0_c4x64.md).  A lane whose stamp misses the block at its own channel reads
// zeros from the padded kernel table, so there is no divergence in the FMA body at all.
//
//   A1 (thread = candidate row, once per super-group): walk the uv buckets (k_bin.cu) that can reach the tile
//       at ANY scale of the 192 channels, keep the rows whose stamp can overlap the tile (conservative fp64
//       interval test).  Then, per 32-channel group:
//   F  (thread = list entry, once per super-group): the same test against each group's own scale range, from
//       shared memory -> one selection per group.  Compaction is by ballot + prefix in both steps, so the hit
//       order is a pure function of the sorted rows.
//   A2 (warp = hit, lane = channel): cp.async of the hit's 32 visibilities (1 KB) and weights into shared
//       memory; while they fly, the exact index function (index.cuh) per (row, channel) gives the lane a packed
//       pair of kernel-table offsets ("geo") and the hit a bit mask of the blocks any lane touches.
//   B  (warp = block, lane = channel): for every hit that touches the block: 2 x LDS.128 of V, one LDS of w
//       (folded into the two v taps), LDS.128 + LDS.64 of kernel taps from shifted zero-padded table copies,
//       8 FMUL, 32 FFMA2 (fma.rn.f32x2); software-pipelined over two register sets.
//   write-out: registers -> padded shared-memory stage (aliasing the w*V batch) -> full 128 B lines of one
//       (channel, pol, row) with streaming stores; every cell of grid_out is written exactly once, zeros
//       included (R10).
//
// No atomics on grid data, no fp64 and no global loads in phase B.  A tile too dense for the list is served by
// resumable A1 sweeps per group.  Two co-resident CTAs hide part of each other's barriers and load latency.
// Tiles are walked row-major (neighbouring tiles share visibility rows in L2), super-groups fastest.
#include "plan.h"

namespace mwa {

constexpr int kcWarps = 8;
constexpr int kcThreads = kcWarps * 32;
constexpr int kcLanes = 32;            // channels per group
constexpr int kcSuper = 6;             // groups per super-group (one A1 sweep serves them all)
constexpr int kcTileX = 16, kcTileY = 4;
constexpr int kcListCap = 640;         // candidate hits kept per A1 sweep chunk (row id + uv)
constexpr int kcBatch = 64;            // hits per A2/B batch (w*V: 64 KB, geo: 8 KB)
constexpr int kcGroupCap = 32;         // channel groups whose scale table is cached in shared memory (1024 channels)
constexpr int kcPadU = 20;             // zero padding (floats) in front of a u table row
constexpr int kcPadV = kcTileY;        // ... of a v table row
constexpr int kcZeroFloats = 32;       // all-zero block behind each table (target of an invalid lane's geo)
constexpr int kcChanStride = 4 * kcTileY * 128 + 16;   // stage bytes per channel: 4 pol x 4 rows x 128 B, +16 B so
                                                       // that the 8 lanes of an STS.128 quarter-warp hit all 32 banks
constexpr int kcStageBytes = kcLanes * kcChanStride;   // 66,048 B >= the 65,536 B of a w*V batch

struct ChanParams {
    GridGeom g;
    const double* scale;        // [n_chan]
    const double4* group;       // [n_groups] s_lo, s_hi, s_ref / s_lo, s_ref / s_hi (scale_kernel)
    const int* bucket_start;    // [nb*nb + 1]
    const double4* row_sorted;  // [n_vis] (u, v, row id, 0) of the bucket-sorted rows
    int* counter;               // work counter
    int* stats;                 // diagnostics (mwa_grid_plan_last_stats): [6] items served by the dense path
    const int* dispatch;        // device-side design choice (AUTO): run only if *dispatch == dispatch_want; null = always
    int dispatch_want;
    const float4* vis;          // [n_vis][n_chan][2] float4
    const float* weights;       // [n_vis][n_chan] or null
    const float* table;         // [(O+1)][W]
    float* grid;                // [n_chan][4][N][N][2]
    int n_chan, n_groups, nb, nt;
    int rlu, rlv;               // padded row lengths of the shifted table copies
    int n_tu, n_tv;             // floats in the u / v table copies (zero blocks excluded)
    int n_items;
    double reach;               // h + 1/2 + 1/(2O) + eps: |x - ic| <= 1/2 + 1/(2O) by construction of INDEX (R4)
};

typedef unsigned long long u64;

__device__ __forceinline__ void c_unpack2(u64 v, float& a, float& b) {
    asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v));
}
__device__ __forceinline__ u64 c_pack2(float a, float b) {
    u64 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b));
    return r;
}
__device__ __forceinline__ void c_ffma2(u64& d, u64 a, u64 b) {       // d = a * b + d on two fp32 lanes
    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(d) : "l"(a), "l"(b));
}
__device__ __forceinline__ void c_st_stream_v4(float* p, float4 v) {
    asm volatile("st.global.cs.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}


struct ChanSmem {                 // fixed part; the table copies follow it in dynamic shared memory
    __align__(16) unsigned char zs[kcStageBytes];   // w*V of the batch [hit][lane][8 floats]; aliased by the write-out stage
    unsigned geo[kcBatch * kcLanes];
    float wts[kcBatch * kcLanes];                   // weights of the batch [hit][lane] (cp.async target)
    double2 hit_uv[kcListCap];                      // the list: uv (metres) and original row of each candidate hit
    int hit_row[kcListCap];
    unsigned short sel[kcSuper][kcListCap];         // per group of the super-group: the list entries that reach the tile, in list order
    int sel_cnt[kcSuper];
    unsigned hit_mask[kcBatch];
    unsigned char vlist[kcWarps][kcBatch];          // per warp: the batch hits that touch its block, in order
    unsigned char lut_u[32], lut_v[32];             // block masks by stamp origin: [ou + W - 1] -> bx bits, [ov + W - 1] -> by bits (x16)
    int warp_cnt[2][kcSuper][kcWarps];
    int next_item;
    double4 group[kcGroupCap];                      // copy of the per-group scale table (scale_kernel)
    double sc[kcSuper][kcLanes];                    // channel scales s_c of the current super-group
};

template <bool HAS_W>
__global__ void __launch_bounds__(kcThreads, 2)
chan_kernel(const __grid_constant__ ChanParams P) {
    if (P.dispatch != nullptr && *P.dispatch != P.dispatch_want) return;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    ChanSmem& S = *reinterpret_cast<ChanSmem*>(smem_raw);
    float* tu = reinterpret_cast<float*>(smem_raw + ((sizeof(ChanSmem) + 15) & ~size_t(15)));
    float* tv = tu + P.n_tu + kcZeroFloats;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int W = P.g.W, O1 = P.g.O + 1, N = P.g.N, hW = P.g.h;

    // ---- shifted, zero-padded kernel-table copies (once per CTA)
    //   tu[s][r][q] = Tp_u[r][q + s], Tp_u[r][kcPadU + t] = T[r][t]     s = 0..3  (LDS.128 alignment)
    //   tv[s][r][q] = Tp_v[r][q + s], Tp_v[r][kcPadV + t] = T[r][t]     s = 0..1  (LDS.64 alignment)
    for (int k = tid; k < P.n_tu + kcZeroFloats; k += kcThreads) {
        float v = 0.0f;
        if (k < P.n_tu) {
            const int q = k % P.rlu, r = (k / P.rlu) % O1, s = k / (P.rlu * O1);
            const int t = q + s - kcPadU;
            if (t >= 0 && t < W) v = P.table[r * W + t];
        }
        tu[k] = v;
    }
    for (int k = tid; k < P.n_tv + kcZeroFloats; k += kcThreads) {
        float v = 0.0f;
        if (k < P.n_tv) {
            const int q = k % P.rlv, r = (k / P.rlv) % O1, s = k / (P.rlv * O1);
            const int t = q + s - kcPadV;
            if (t >= 0 && t < W) v = P.table[r * W + t];
        }
        tv[k] = v;
    }
    if (tid < 32) {                                                  // W <= 15: ou + W - 1 <= 29, ov + W - 1 <= 17
        const int ou = tid - (W - 1);
        unsigned mu = 0u, mv = 0u;
        if (ou < kcTileX) {
            const int bxl = max(0, ou >> 2), bxh = min(kcTileX / 4 - 1, (ou + W - 1) >> 2);
            mu = (2u << bxh) - (1u << bxl);
        }
        if (ou < kcTileY) {                                           // same index reused as ov
            const int bl = max(0, ou >> 1), bh = min(kcTileY / 2 - 1, (ou + W - 1) >> 1);
            for (int b = bl; b <= bh; ++b) mv |= 1u << (4 * b);
        }
        S.lut_u[tid] = (unsigned char)mu;
        S.lut_v[tid] = (unsigned char)mv;
    }
    for (int k = tid; k < min(P.n_groups, kcGroupCap); k += kcThreads) S.group[k] = P.group[k];
    const double4* group = P.n_groups <= kcGroupCap ? S.group : P.group;
    const int n_sg = (P.n_groups + kcSuper - 1) / kcSuper;
    if (tid == 0) S.next_item = atomicAdd(P.counter, 1);
    __syncthreads();

    const int bx = warp & 3, by = warp >> 2;
    const unsigned wbit = (unsigned)warp;                            // bit by * 4 + bx of a hit mask
    const unsigned tu_s = (unsigned)__cvta_generic_to_shared(tu) + 16u * bx;
    const unsigned tv_s = (unsigned)__cvta_generic_to_shared(tv) + 8u * by;
    const unsigned zs_s = (unsigned)__cvta_generic_to_shared(S.zs) + 32u * lane;
    const unsigned geo_s = (unsigned)__cvta_generic_to_shared(S.geo) + 4u * lane;
    const unsigned wt_s = (unsigned)__cvta_generic_to_shared(S.wts) + 4u * lane;
    const unsigned zero_geo = (unsigned)(P.n_tu * 4) | ((unsigned)(P.n_tv * 4) << 16);
    const size_t plane = (size_t)N * N;
    const unsigned lt_mask = (1u << lane) - 1u;
    const unsigned full = 0xffffffffu;


    int item = S.next_item;
    while (item < P.n_items) {
        int next_item = 0;
        if (tid == 0) next_item = atomicAdd(P.counter, 1);           // latency hidden behind this item
        const int sgi = item % n_sg;
        const int ts = item / n_sg;
        const int tile = ts >> 2;                                    // row-major over the 16x16 super-tiles: neighbours in time share visibility rows in L2
        if (warp < kcSuper)      // channel scales of the super-group; visible after the barriers of the sweep
            S.sc[warp][lane] = P.scale[min((sgi * kcSuper + warp) * kcLanes + lane, P.n_chan - 1)];
        const int ty = tile / P.nt, tx = tile - ty * P.nt;
        const int X0 = tx * kcTileX, Y0 = ty * 16 + (ts & 3) * kcTileY;
        if (Y0 < N) {
            // per-group state (set in the group loop below, captured by reference)
            int c0 = 0, cc = 0, gslot = 0;
            const unsigned short* sel = S.sel[0];                        // selection in use (group slot, or slot 0 after a dense sweep)
            bool cvalid = false;
            u64 acc[2][4][4];   // [row i][col j][pol] = (re, im) of the lane's channel

            // ---- A2: n hits starting at selection entry b0, warp = hit, lane = channel
            auto phase_a2 = [&](int b0, int n) {
                // (i) cp.async the warp's visibilities (32 lanes x 32 B = 1 KB per hit) and weights straight into
                //     shared memory: every copy of the batch is in flight while (ii) does the fp64 index work
                for (int hh = warp; hh < n; hh += kcWarps) {
                    const size_t sidx = (size_t)S.hit_row[sel[b0 + hh]] * P.n_chan + cc;
                    const float4* src = P.vis + 2 * sidx;
                    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(zs_s + 1024u * hh), "l"(src) : "memory");
                    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(zs_s + 1024u * hh + 16u), "l"(src + 1) : "memory");
                    if (HAS_W)
                        asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(wt_s + 128u * hh), "l"(P.weights + sidx) : "memory");
                }
                asm volatile("cp.async.commit_group;" ::: "memory");
                // (ii) exact indices -> geo, block mask
                const double sc = S.sc[gslot][lane];
                unsigned dropped = 0u;                                             // bit k: this lane's sample of hit warp + k * kcWarps is dropped (R11)
#pragma unroll 2
                for (int hh = warp; hh < n; hh += kcWarps) {
                    const double2 p = S.hit_uv[sel[b0 + hh]];
                    SampleIndex s;
                    unsigned geo = zero_geo, mask = 0u;
                    const bool valid = sample_index(p.x, p.y, sc, P.g, s) && cvalid;
                    if (!valid) dropped |= 1u << (hh / kcWarps);
                    if (valid) {
                        const int tu_ = kcPadU + hW + X0 - s.iu, tv_ = kcPadV + hW + Y0 - s.iv;   // pad - (stamp origin relative to the tile)
                        const unsigned iu_ = (unsigned)(kcPadU + W - 1 - tu_), iv_ = (unsigned)(kcPadV + W - 1 - tv_);   // ou + W - 1, ov + W - 1
                        if (iu_ < (unsigned)(kcTileX + W - 1) && iv_ < (unsigned)(kcTileY + W - 1)) {
                            const int su = tu_ & 3, sv = tv_ & 1;
                            const int offu = s.ru * P.rlu + tu_ + su * (O1 * P.rlu - 1);
                            const int offv = s.rv * P.rlv + tv_ + sv * (O1 * P.rlv - 1);
                            geo = (unsigned)(offu * 4) | ((unsigned)(offv * 4) << 16);
                            mask = (unsigned)S.lut_v[iv_] * (unsigned)S.lut_u[iu_];
                        }
                    }
                    mask = __reduce_or_sync(full, mask);                           // blocks touched by any lane
                    asm volatile("st.shared.u32 [%0], %1;" ::"r"(geo_s + 128u * hh), "r"(geo) : "memory");
                    if (lane == 0) S.hit_mask[hh] = mask;
                }
                asm volatile("cp.async.wait_group 0;" ::: "memory");              // visible to the other warps after the barrier
                // a dropped sample contributes nothing, whatever its visibility holds (a flagged NaN times a zero tap would
                // still be NaN): its staged visibility is overwritten with zeros.  Rare: only samples at the grid edge.
                for (; dropped != 0u; dropped &= dropped - 1u) {
                    const unsigned hh = (unsigned)warp + (unsigned)(__ffs(dropped) - 1) * kcWarps;
                    asm volatile("st.shared.v4.f32 [%0], {%1, %1, %1, %1};" ::"r"(zs_s + 1024u * hh), "f"(0.0f) : "memory");
                    asm volatile("st.shared.v4.f32 [%0], {%1, %1, %1, %1};" ::"r"(zs_s + 1024u * hh + 16u), "f"(0.0f) : "memory");
                    if (HAS_W) asm volatile("st.shared.f32 [%0], %1;" ::"r"(wt_s + 128u * hh), "f"(0.0f) : "memory");
                }
            };

            // ---- B: the warp's block against the n hits of the batch; every lane computes, zeros where it misses
            auto phase_b = [&](int n) {
                int cnt = 0;
#pragma unroll
                for (int gq = 0; gq < kcBatch / 32; ++gq) {
                    if (gq * 32 < n) {
                        const int idx = gq * 32 + lane;
                        const unsigned hm = idx < n ? S.hit_mask[idx] : 0u;
                        const bool t = (hm >> wbit) & 1u;
                        const unsigned m = __ballot_sync(full, t);
                        if (t) S.vlist[warp][cnt + __popc(m & lt_mask)] = (unsigned char)idx;
                        cnt += __popc(m);
                    }
                }
                __syncwarp();
                if (cnt == 0) return;
                // software pipeline, two visits per trip with two register sets (no rotation moves): the taps, the
                // weight and the visibility of visit v+1 and the geo of visit v+2 are loaded while the 32 FFMA2 of
                // visit v issue, so no LDS latency is exposed inside the loop
                const unsigned char* vl = S.vlist[warp];
                const int last = cnt - 1;
#define K5_LOAD(h, g, Z0, Z1, Z2, Z3, U0, U1, U2, U3, V0, V1, WT)                                                         \
    asm volatile("ld.shared.v2.b64 {%0, %1}, [%2];" : "=l"(Z0), "=l"(Z1) : "r"(zs_s + 1024u * (h)));                       \
    asm volatile("ld.shared.v2.b64 {%0, %1}, [%2];" : "=l"(Z2), "=l"(Z3) : "r"(zs_s + 1024u * (h) + 16u));                 \
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(U0), "=f"(U1), "=f"(U2), "=f"(U3) : "r"(tu_s + ((g) & 0xffffu))); \
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(V0), "=f"(V1) : "r"(tv_s + ((g) >> 16)));                       \
    if (HAS_W) asm volatile("ld.shared.f32 %0, [%1];" : "=f"(WT) : "r"(wt_s + 128u * (h)));
#define K5_FMA(Z0, Z1, Z2, Z3, U0, U1, U2, U3, V0, V1, WT)                                                                \
    {                                                                                                                     \
        const float kvw[2] = {HAS_W ? V0 * WT : V0, HAS_W ? V1 * WT : V1};                                                \
        const float kuu[4] = {U0, U1, U2, U3};                                                                            \
        _Pragma("unroll") for (int i = 0; i < 2; ++i) _Pragma("unroll") for (int j = 0; j < 4; ++j) {                      \
            const float k = kvw[i] * kuu[j];                                                                              \
            const u64 kk = c_pack2(k, k);                                                                                 \
            c_ffma2(acc[i][j][0], kk, Z0);                                                                                \
            c_ffma2(acc[i][j][1], kk, Z1);                                                                                \
            c_ffma2(acc[i][j][2], kk, Z2);                                                                                \
            c_ffma2(acc[i][j][3], kk, Z3);                                                                                \
        }                                                                                                                 \
    }
                u64 az0, az1, az2, az3, bz0, bz1, bz2, bz3;
                float au0, au1, au2, au3, av0, av1, aw = 1.0f, bu0, bu1, bu2, bu3, bv0, bv1, bw = 1.0f;
                unsigned h1 = vl[min(1, last)], h2 = vl[min(2, last)], g1, g2;
                {
                    const unsigned h0 = vl[0];
                    unsigned g0;
                    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(g0) : "r"(geo_s + 128u * h0));
                    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(g1) : "r"(geo_s + 128u * h1));
                    K5_LOAD(h0, g0, az0, az1, az2, az3, au0, au1, au2, au3, av0, av1, aw)
                }
#pragma unroll 1
                for (int v = 0; v < cnt; v += 2) {
                    // set B <- visit v+1 ; geo of v+2 ; then FMAs of visit v from set A
                    K5_LOAD(h1, g1, bz0, bz1, bz2, bz3, bu0, bu1, bu2, bu3, bv0, bv1, bw)
                    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(g2) : "r"(geo_s + 128u * h2));
                    const unsigned h3 = vl[min(v + 3, last)];
                    K5_FMA(az0, az1, az2, az3, au0, au1, au2, au3, av0, av1, aw)
                    if (v + 1 >= cnt) break;
                    // set A <- visit v+2 ; geo of v+3 ; then FMAs of visit v+1 from set B
                    K5_LOAD(h2, g2, az0, az1, az2, az3, au0, au1, au2, au3, av0, av1, aw)
                    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(g1) : "r"(geo_s + 128u * h3));
                    const unsigned h4 = vl[min(v + 4, last)];
                    K5_FMA(bz0, bz1, bz2, bz3, bu0, bu1, bu2, bu3, bv0, bv1, bw)
                    h1 = h3;
                    h2 = h4;
                }
#undef K5_LOAD
#undef K5_FMA
            };

            // the first n selection entries, in batches: A2 | sync | B | sync
            auto process_sel = [&](int n) {
                for (int b0 = 0; b0 < n; b0 += kcBatch) {
                    const int nbat = min(kcBatch, n - b0);
                    phase_a2(b0, nbat);
                    __syncthreads();
                    phase_b(nbat);
                    __syncthreads();
                }
            };

            int par = 0;                                                   // parity of the warp_cnt buffer in use
            // deterministic CTA-wide compaction step for up to kcSuper independent selections at once: slot[q] receives
            // the slot of this thread's hit in selection q (or -1) and count[q] grows by the chunk's hits; ONE __syncthreads
            auto compact = [&](const bool (&hit)[kcSuper], int nq, int (&count)[kcSuper], int (&slot)[kcSuper]) {
                unsigned ball[kcSuper];
#pragma unroll
                for (int q = 0; q < kcSuper; ++q) {
                    ball[q] = q < nq ? __ballot_sync(full, hit[q]) : 0u;
                    if (lane == 0 && q < nq) S.warp_cnt[par][q][warp] = __popc(ball[q]);
                }
                __syncthreads();
#pragma unroll
                for (int q = 0; q < kcSuper; ++q) {
                    slot[q] = -1;
                    if (q < nq) {
                        const int cv = lane < kcWarps ? S.warp_cnt[par][q][lane] : 0;
                        int ci = cv;
#pragma unroll
                        for (int o = 1; o < kcWarps; o <<= 1) {
                            const int t = __shfl_up_sync(full, ci, o);
                            if (lane >= o) ci += t;
                        }
                        const int tot = __shfl_sync(full, ci, kcWarps - 1);
                        const int wbase = __shfl_sync(full, ci - cv, warp);
                        if (hit[q]) slot[q] = count[q] + wbase + __popc(ball[q] & lt_mask);
                        count[q] += tot;
                    }
                }
                par ^= 1;
            };
            auto reaches_tile = [&](const double2 p, double s_lo, double s_hi) -> bool {
                const double halfN = (double)(N / 2);
                const double cx0 = (double)X0 - halfN, cx1 = (double)(X0 + kcTileX - 1) - halfN;
                const double cy0 = (double)Y0 - halfN, cy1 = (double)(Y0 + kcTileY - 1) - halfN;
                const double xa = __dmul_rn(__dmul_rn(p.x, s_lo), P.g.inv_du), xb = __dmul_rn(__dmul_rn(p.x, s_hi), P.g.inv_du);
                const double ya = __dmul_rn(__dmul_rn(p.y, s_lo), P.g.inv_du), yb = __dmul_rn(__dmul_rn(p.y, s_hi), P.g.inv_du);
                return fmax(xa, xb) + P.reach >= cx0 && fmin(xa, xb) - P.reach <= cx1 &&
                       fmax(ya, yb) + P.reach >= cy0 && fmin(ya, yb) - P.reach <= cy1;
            };

            // ---- A1: bucket sweep for scales in [s_lo, s_hi] (il, ih = s_ref / s_lo, s_ref / s_hi, NaN = scan all buckets).
            // Resumable: fills the list (identity selection in sel slot 0) from position (rg, base) of the scan until the
            // next chunk of kcThreads candidates might not fit, and returns the number of entries; done = scan finished.
            auto sweep = [&](double s_lo, double s_hi, double il, double ih, int& rg, int& base, bool& done) -> int {
                int wx0 = 0, wx1 = P.nb - 1, wy0 = 0, wy1 = P.nb - 1;
                if (il == il && ih == ih) {
                    const double halfN = (double)(N / 2);
                    const double cx0 = (double)X0 - halfN, cx1 = (double)(X0 + kcTileX - 1) - halfN;
                    const double cy0 = (double)Y0 - halfN, cy1 = (double)(Y0 + kcTileY - 1) - halfN;
                    const double pad = (double)hW + 1.25;
                    const double ax = cx0 - pad, bxx = cx1 + pad, ay = cy0 - pad, byy = cy1 + pad;
                    const double ib = 1.0 / kBucketCells, top = (double)(P.nb - 1);
                    wx0 = (int)fmin(fmax(floor((fmin(ax * il, ax * ih) + halfN) * ib), 0.0), top);
                    wx1 = (int)fmin(fmax(floor((fmax(bxx * il, bxx * ih) + halfN) * ib), 0.0), top);
                    wy0 = (int)fmin(fmax(floor((fmin(ay * il, ay * ih) + halfN) * ib), 0.0), top);
                    wy1 = (int)fmin(fmax(floor((fmax(byy * il, byy * ih) + halfN) * ib), 0.0), top);
                }
                if (rg < 0) { rg = wy0; base = 0; }
                int count[kcSuper] = {};
                bool full_list = false;
                for (; rg <= wy1 && !full_list; rg += 32, base = 0) {
                    int k0 = 0, len = 0;
                    if (rg + lane <= wy1) {
                        k0 = __ldg(P.bucket_start + (rg + lane) * P.nb + wx0);
                        len = __ldg(P.bucket_start + (rg + lane) * P.nb + wx1 + 1) - k0;
                    }
                    int incl = len;
#pragma unroll
                    for (int o = 1; o < 32; o <<= 1) {
                        const int t = __shfl_up_sync(full, incl, o);
                        if (lane >= o) incl += t;
                    }
                    const int total = __shfl_sync(full, incl, 31);
                    const int excl = incl - len;
                    for (; base < total; base += kcThreads) {
                        if (count[0] + kcThreads > kcListCap) { full_list = true; break; }   // uniform; resume here next time
                        const int f = base + tid;
                        bool hit[kcSuper] = {};
                        double2 p = make_double2(0.0, 0.0);
                        int k = 0;
                        {
                            int lo = 0;                                         // smallest r with incl[r] > f
#pragma unroll
                            for (int st = 16; st > 0; st >>= 1) {
                                const int t = __shfl_sync(full, incl, lo + st - 1);
                                if (t <= f) lo += st;
                            }
                            lo = min(lo, 31);
                            const int rk0 = __shfl_sync(full, k0, lo), rex = __shfl_sync(full, excl, lo);
                            k = rk0 + (f - rex);
                        }
                        double rowd = 0.0;
                        if (f < total) {
                            const double4 rec = P.row_sorted[k];
                            p = make_double2(rec.x, rec.y);
                            rowd = rec.z;
                            hit[0] = reaches_tile(p, s_lo, s_hi);
                        }
                        int slot[kcSuper];
                        compact(hit, 1, count, slot);
                        if (slot[0] >= 0) {
                            S.hit_uv[slot[0]] = p;
                            S.hit_row[slot[0]] = (int)rowd;
                            S.sel[0][slot[0]] = (unsigned short)slot[0];
                        }
                    }
                    if (full_list) break;                                      // keep rg and base for the resume
                }
                done = !full_list;
                __syncthreads();                                           // list complete and visible
                return count[0];
            };

            // ---- a5: write the lane-channel tiles of the current group, once (zeros when nothing reached the tile)
            auto write_out = [&](bool any) {
                if (any) {
#pragma unroll
                    for (int pol = 0; pol < 4; ++pol)
#pragma unroll
                        for (int i = 0; i < 2; ++i) {
                            float a0, a1, a2, a3, b0, b1, b2, b3;
                            c_unpack2(acc[i][0][pol], a0, a1); c_unpack2(acc[i][1][pol], a2, a3);
                            c_unpack2(acc[i][2][pol], b0, b1); c_unpack2(acc[i][3][pol], b2, b3);
                            unsigned char* dst = S.zs + lane * kcChanStride + (pol * kcTileY + 2 * by + i) * 128 + bx * 32;
                            *reinterpret_cast<float4*>(dst) = make_float4(a0, a1, a2, a3);
                            *reinterpret_cast<float4*>(dst + 16) = make_float4(b0, b1, b2, b3);
                        }
                    __syncthreads();
                }
                const int j = tid & 7, row = (tid >> 3) & 3, q0 = tid >> 5;       // 16 B chunk, tile row, (channel, pol) slot
                const int y = Y0 + row, x = X0 + 2 * j, pol = q0 & 3;
                if (y < N && x < N) {
                    const unsigned char* src = S.zs + (q0 >> 2) * kcChanStride + (pol * kcTileY + row) * 128 + j * 16;
                    float* dst = P.grid + (((size_t)(c0 + (q0 >> 2)) * 4 + pol) * plane + (size_t)y * N + x) * 2;
                    const int nch = min(kcLanes, P.n_chan - c0);
#pragma unroll 8
                    for (int ch = q0 >> 2; ch < nch; ch += 2) {
                        float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
                        if (any) v = *reinterpret_cast<const float4*>(src);
                        c_st_stream_v4(dst, v);
                        src += 2 * kcChanStride;
                        dst += 2 * 4 * plane * 2;
                    }
                }
                // the stage aliases the visibility batch: nobody may start the next group's cp.async (A2) while a slower
                // warp is still copying this group's stage out
                if (any) __syncthreads();
            };

            // ---- the super-group: one sweep over the union of its groups' scale ranges ...
            const int g_begin = sgi * kcSuper, g_end = min(P.n_groups, g_begin + kcSuper);
            double u_lo = 0.0, u_hi = 0.0, u_il = 0.0, u_ih = 0.0;
            for (int g = g_begin; g < g_end; ++g) {
                const double4 gi = group[g];
                if (g == g_begin) { u_lo = gi.x; u_hi = gi.y; u_il = gi.z; u_ih = gi.w; }
                else {
                    u_lo = fmin(u_lo, gi.x); u_hi = fmax(u_hi, gi.y);
                    u_il = (gi.z == gi.z && u_il == u_il) ? fmax(u_il, gi.z) : gi.z + u_il;      // NaN is sticky
                    u_ih = (gi.w == gi.w && u_ih == u_ih) ? fmin(u_ih, gi.w) : gi.w + u_ih;
                }
            }
            int rg = -1, base = 0;
            bool done = false;
            int n_super = 0;
            if (g_end - g_begin > 1) n_super = sweep(u_lo, u_hi, u_il, u_ih, rg, base, done);
            const bool dense = !done;                                      // list too small for the tile (or a single group)
            if (dense && tid == 0) atomicAdd(P.stats + 6, 1);

            // ... F: one pass over the list selects, for every group of the super-group, the entries that reach the tile
            if (!dense) {
                const int nq = g_end - g_begin;
                int count[kcSuper] = {};
                for (int b0 = 0; b0 < n_super; b0 += kcThreads) {
                    const int i = b0 + tid;
                    bool hit[kcSuper] = {};
                    if (i < n_super) {
                        const double2 p = S.hit_uv[i];
#pragma unroll
                        for (int q = 0; q < kcSuper; ++q)
                            if (q < nq) hit[q] = reaches_tile(p, group[g_begin + q].x, group[g_begin + q].y);
                    }
                    int slot[kcSuper];
                    compact(hit, nq, count, slot);
#pragma unroll
                    for (int q = 0; q < kcSuper; ++q)
                        if (slot[q] >= 0) S.sel[q][slot[q]] = (unsigned short)i;
                }
                if (tid == 0) {
#pragma unroll
                    for (int q = 0; q < kcSuper; ++q) S.sel_cnt[q] = count[q];
                }
                __syncthreads();
            }

            // ... then group by group: A2 + B over the selection (or, for a dense tile, over resumable sweeps), write
            for (int g = g_begin; g < g_end; ++g) {
                c0 = g * kcLanes;
                gslot = g - g_begin;
                cvalid = c0 + lane < P.n_chan;
                cc = cvalid ? c0 + lane : P.n_chan - 1;
                sel = dense ? S.sel[0] : S.sel[gslot];
#pragma unroll
                for (int i = 0; i < 2; ++i)
#pragma unroll
                    for (int j = 0; j < 4; ++j)
#pragma unroll
                        for (int p = 0; p < 4; ++p) acc[i][j][p] = 0ull;
                bool any = false, more = true;
                rg = -1;
                while (more) {
                    int n;
                    if (dense) {
                        const double4 gi = group[g];
                        bool fin = false;
                        n = sweep(gi.x, gi.y, gi.z, gi.w, rg, base, fin);
                        more = !fin;
                    } else {
                        n = S.sel_cnt[gslot];
                        more = false;
                    }
                    if (n > 0) {
                        process_sel(n);                                        // the only call site: A2 | sync | B | sync per batch
                        any = true;
                    }
                }
                write_out(any);
            }
        }   // Y0 < N
        __syncthreads();
        if (tid == 0) S.next_item = next_item;
        __syncthreads();
        item = S.next_item;
    }
}

// Geometry of the padded table copies (see the kernel header).
static void chan_table_geometry(const GridGeom& g, ChanParams& P) {
    P.rlu = (g.W + 35 + 3) & ~3;              // kcPadU + (W - 1) + 12 + 4, rounded up to a multiple of 4
    P.rlv = 2 * kcTileY + g.W + 1;            // even because W is odd
    P.n_tu = 4 * (g.O + 1) * P.rlu;
    P.n_tv = 2 * (g.O + 1) * P.rlv;
}

static size_t chan_smem_bytes(const ChanParams& P) {
    return ((sizeof(ChanSmem) + 15) & ~size_t(15)) + (size_t)(P.n_tu + P.n_tv + 2 * kcZeroFloats) * sizeof(float);
}

bool chan_supported(const Plan* p, int n_chan) {
    if (n_chan < 1) return false;
    ChanParams P;
    chan_table_geometry(p->geom, P);
    if ((P.n_tu + kcZeroFloats) * 4 > 65535 || (P.n_tv + kcZeroFloats) * 4 > 65535) return false;   // geo packs 16-bit byte offsets
    return chan_smem_bytes(P) <= 227 * 1024;
}

bool launch_chan(Plan* p, const float* vis, const float* w, long long n_vis, int n_chan, float* grid,
                 const int* dispatch, cudaStream_t st) {
    (void)n_vis;
    if (!chan_supported(p, n_chan)) { set_error("design CHAN does not support this kernel table size"); return false; }
    ChanParams P;
    P.g = p->geom;
    chan_table_geometry(p->geom, P);
    P.scale = p->ws.d_scale;
    P.group = (const double4*)p->ws.d_group;
    P.bucket_start = p->ws.d_bucket_count;
    P.row_sorted = (const double4*)p->ws.d_row_sorted;
    P.counter = p->ws.d_misc + 1;
    P.stats = p->ws.d_misc + 4;
    P.dispatch = dispatch;
    P.dispatch_want = 1;
    P.vis = (const float4*)vis;
    P.weights = w;
    P.table = p->d_table;
    P.grid = grid;
    P.n_chan = n_chan;
    P.n_groups = (n_chan + kcLanes - 1) / kcLanes;
    P.nb = (p->geom.N + kBucketCells - 1) / kBucketCells;
    P.nt = (p->geom.N + kTile - 1) / kTile;
    P.reach = (double)p->geom.h + 0.5 + 0.5 / (double)p->geom.O + 1e-6;
    const int n_sg = (P.n_groups + kcSuper - 1) / kcSuper;
    const long long n_items = (long long)P.nt * P.nt * (16 / kcTileY) * n_sg;
    if (n_items >= 0x7fffffffLL) { set_error("design CHAN: too many work items"); return false; }
    P.n_items = (int)n_items;
    const size_t smem = chan_smem_bytes(P);
    auto kern = w ? chan_kernel<true> : chan_kernel<false>;
    // a per-device setting: set on every launch (cheap)
    if (!cuda_ok(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024), "chan smem attribute"))
        return false;
    int ctas_per_sm = 0;
    if (!cuda_ok(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&ctas_per_sm, kern, kcThreads, smem), "chan occupancy"))
        return false;
    if (ctas_per_sm < 1) { set_error("chan kernel does not fit on an SM"); return false; }
    long long blocks = (long long)p->sm_count * ctas_per_sm;
    if (blocks > n_items) blocks = n_items;
    if (blocks < 1) blocks = 1;
    kern<<<(unsigned)blocks, kcThreads, smem, st>>>(P);
    p->last_launches += 1;
    return cuda_ok(cudaGetLastError(), "chan_kernel");
}

}  // namespace mwa
