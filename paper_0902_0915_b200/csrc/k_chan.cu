// k_chan.cu - K5, the channel-SIMD register gridder (a2 + a4 + a5 fused) for finely channelised data.
//
// The correlator of PAPER.md:19 delivers 768 channels of 40 kHz: neighbouring channels see the same baseline
// at almost the same (u, v) (u_lambda = u_m * nu / c moves by 2.6e-4 of its radius per channel), and every
// channel owns its own grid (BASELINE.json configs[3]).  K5 turns that into SIMD lanes:
//
//   CTA  = one 16 x 8 cell tile  x  one group of 32 adjacent channels (all 4 polarisations); 16 warps
//   warp = one 4x2-cell block of the tile
//   lane = one channel of the group; the lane keeps 8 cells x 4 pol x (re, im) = 64 fp32 accumulators
//          of ITS channel's grid in registers.
//
// All 32 lanes of a warp therefore walk (almost) the same list of baseline rows - the walk is balanced by
// construction, where K3c (k_gather.cu: lane = block, same channel) leaves 23 of 32 lanes idle on Poisson
// noise (profiles/r01_gather_v0_c4x64.md).  A lane whose stamp misses the block at its own channel reads
// zeros from the padded kernel table, so there is no divergence in the FMA body at all.
//
//   A1 (thread = candidate row): walk the uv buckets (k_bin.cu) that can reach the tile at ANY scale of the
//       channel group, keep the rows whose stamp can overlap the tile (conservative fp64 interval test);
//       compaction is by ballot + prefix, so the hit order - and with it every fp32 sum - is deterministic.
//   A2 (warp = hit, lane = channel): coalesced load of the hit's 32 visibilities (1 KB) and weights, w*V
//       staged in shared memory; the exact index function (index.cuh) per (row, channel) gives the lane a
//       packed pair of kernel-table offsets ("geo"); per hit a bit mask of the blocks any lane touches.
//   B  (warp = block, lane = channel): for every hit that touches the block: 2 x LDS.128 of w*V, LDS.128 +
//       LDS.64 of kernel taps from shifted zero-padded table copies, 8 FMUL, 32 FFMA2 (fma.rn.f32x2).
//   write-out: registers -> padded shared-memory stage (aliasing the w*V batch) -> full 128 B lines of one
//       (channel, pol, row) with streaming stores; every cell of grid_out is written exactly once, zeros
//       included (R10).
//
// No atomics on grid data, no fp64 in phase B, no global loads in phase B.
#include "plan.h"

namespace mwa {

constexpr int kcWarps = 16;
constexpr int kcThreads = kcWarps * 32;
constexpr int kcLanes = 32;            // channels per group
constexpr int kcTileX = 16, kcTileY = 8;
constexpr int kcListCap = 1024;        // candidate hits kept per A1 sweep (row id + uv)
constexpr int kcBatch = 128;           // hits per A2/B batch (w*V: 128 KB, geo: 16 KB)
constexpr int kcPadU = 20;             // zero padding (floats) in front of a u table row
constexpr int kcPadV = kcTileY;        // ... of a v table row
constexpr int kcZeroFloats = 32;       // all-zero block behind each table (target of an invalid lane's geo)
constexpr int kcChanStride = 4 * kcTileY * 128 + 16;   // stage bytes per channel: 4 pol x 8 rows x 128 B, +16 B so
                                                       // that the 8 lanes of an STS.128 quarter-warp hit all 32 banks
constexpr int kcStageBytes = kcLanes * kcChanStride;   // 131,584 B >= the 131,072 B of a w*V batch

struct ChanParams {
    GridGeom g;
    const double* scale;        // [n_chan]
    const double* scale_ref;    // [1]
    const int* bucket_start;    // [nb*nb + 1]
    const int* perm;            // [n_vis]
    const double2* uv_sorted;   // [n_vis]
    const int* tile_order;      // [nt*nt] 16x16 super-tiles, heaviest first
    int* counter;               // work counter
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
    double2 hit_uv[kcListCap];
    int hit_row[kcListCap];
    unsigned hit_mask[kcBatch];
    unsigned char vlist[kcWarps][kcBatch];          // per warp: the batch hits that touch its block, in order
    int warp_cnt[2][kcWarps];
    int next_item;
};

template <bool HAS_W>
__global__ void __launch_bounds__(kcThreads, 1)
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
    if (tid == 0) S.next_item = atomicAdd(P.counter, 1);
    __syncthreads();

    const int bx = warp & 3, by = warp >> 2;
    const unsigned wbit = (unsigned)warp;                            // bit by * 4 + bx of a hit mask
    const unsigned tu_s = (unsigned)__cvta_generic_to_shared(tu) + 16u * bx;
    const unsigned tv_s = (unsigned)__cvta_generic_to_shared(tv) + 8u * by;
    const unsigned zs_s = (unsigned)__cvta_generic_to_shared(S.zs) + 32u * lane;
    const unsigned geo_s = (unsigned)__cvta_generic_to_shared(S.geo) + 4u * lane;
    const unsigned zero_geo = (unsigned)(P.n_tu * 4) | ((unsigned)(P.n_tv * 4) << 16);
    const size_t plane = (size_t)N * N;
    const unsigned lt_mask = (1u << lane) - 1u;
    const unsigned full = 0xffffffffu;

    int item = S.next_item;
    while (item < P.n_items) {
        int next_item = 0;
        if (tid == 0) next_item = atomicAdd(P.counter, 1);           // latency hidden behind this item
        const int grp = item % P.n_groups;
        const int ts = item / P.n_groups;
        const int tile = P.tile_order[ts >> 1];
        const int ty = tile / P.nt, tx = tile - ty * P.nt;
        const int X0 = tx * kcTileX, Y0 = ty * 16 + (ts & 1) * kcTileY;
        const int c0 = grp * kcLanes;
        const bool cvalid = c0 + lane < P.n_chan;
        const int cc = cvalid ? c0 + lane : P.n_chan - 1;
        if (Y0 < N) {
            const double sc = P.scale[cc];
            u64 acc[2][4][4];   // [row i][col j][pol] = (re, im) of the lane's channel
#pragma unroll
            for (int i = 0; i < 2; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j)
#pragma unroll
                    for (int p = 0; p < 4; ++p) acc[i][j][p] = 0ull;

            // ---- A2: hits [b0, b0 + n) of the list, warp = hit, lane = channel
            auto phase_a2 = [&](int b0, int n) {
                for (int hh = warp; hh < n; hh += kcWarps) {
                    const double2 p = S.hit_uv[b0 + hh];
                    const size_t sidx = (size_t)S.hit_row[b0 + hh] * P.n_chan + cc;
                    float4 va = __ldg(P.vis + 2 * sidx), vb = __ldg(P.vis + 2 * sidx + 1);
                    float wt = 1.0f;
                    if (HAS_W) wt = __ldg(P.weights + sidx);
                    SampleIndex s;
                    unsigned geo = zero_geo;
                    int ulo = 1 << 20, uhi = -(1 << 20), vlo = 1 << 20, vhi = -(1 << 20);
                    if (cvalid && sample_index(p.x, p.y, sc, P.g, s)) {
                        const int ou = s.iu - hW - X0, ov = s.iv - hW - Y0;        // stamp origin relative to the tile
                        if (ou > -W && ou < kcTileX && ov > -W && ov < kcTileY) {
                            const int su = (kcPadU - ou) & 3, sv = (kcPadV - ov) & 1;
                            const int offu = (su * O1 + s.ru) * P.rlu + (kcPadU - ou - su);
                            const int offv = (sv * O1 + s.rv) * P.rlv + (kcPadV - ov - sv);
                            geo = (unsigned)(offu * 4) | ((unsigned)(offv * 4) << 16);
                            ulo = uhi = ou;
                            vlo = vhi = ov;
                        }
                    }
                    // blocks touched by any lane: bounding box of the lanes' stamps (a superset costs only zeros)
                    ulo = __reduce_min_sync(full, ulo);
                    uhi = __reduce_max_sync(full, uhi);
                    vlo = __reduce_min_sync(full, vlo);
                    vhi = __reduce_max_sync(full, vhi);
                    if (HAS_W) {
                        va.x *= wt; va.y *= wt; va.z *= wt; va.w *= wt;
                        vb.x *= wt; vb.y *= wt; vb.z *= wt; vb.w *= wt;
                    }
                    asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(zs_s + 1024u * hh), "f"(va.x), "f"(va.y), "f"(va.z), "f"(va.w) : "memory");
                    asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(zs_s + 1024u * hh + 16u), "f"(vb.x), "f"(vb.y), "f"(vb.z), "f"(vb.w) : "memory");
                    asm volatile("st.shared.u32 [%0], %1;" ::"r"(geo_s + 128u * hh), "r"(geo) : "memory");
                    if (lane == 0) {
                        unsigned mask = 0u;
                        if (ulo <= uhi) {
                            const int bxl = max(0, ulo >> 2), bxh = min(3, (uhi + W - 1) >> 2);
                            const int bl = max(0, vlo >> 1), bh = min(3, (vhi + W - 1) >> 1);
                            const unsigned m4 = (2u << bxh) - (1u << bxl);
                            const unsigned rows = 0x1111u & (0xFFFFu >> (12 - 4 * bh)) & (0xFFFFu << (4 * bl));
                            mask = rows * m4;
                        }
                        S.hit_mask[hh] = mask;
                    }
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
                unsigned hh = S.vlist[warp][0];
                unsigned geo;
                asm volatile("ld.shared.u32 %0, [%1];" : "=r"(geo) : "r"(geo_s + 128u * hh));
                for (int v = 0; v < cnt; ++v) {
                    const unsigned hn = S.vlist[warp][min(v + 1, cnt - 1)];
                    unsigned geon;
                    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(geon) : "r"(geo_s + 128u * hn));
                    u64 z0, z1, z2, z3;
                    asm volatile("ld.shared.v2.b64 {%0, %1}, [%2];" : "=l"(z0), "=l"(z1) : "r"(zs_s + 1024u * hh));
                    asm volatile("ld.shared.v2.b64 {%0, %1}, [%2];" : "=l"(z2), "=l"(z3) : "r"(zs_s + 1024u * hh + 16u));
                    float ku0, ku1, ku2, ku3, kv0, kv1;
                    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(ku0), "=f"(ku1), "=f"(ku2), "=f"(ku3) : "r"(tu_s + (geo & 0xffffu)));
                    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(kv0), "=f"(kv1) : "r"(tv_s + (geo >> 16)));
                    const float ku[4] = {ku0, ku1, ku2, ku3};
                    const float kv[2] = {kv0, kv1};
#pragma unroll
                    for (int i = 0; i < 2; ++i)
#pragma unroll
                        for (int j = 0; j < 4; ++j) {
                            const float k = kv[i] * ku[j];
                            const u64 kk = c_pack2(k, k);
                            c_ffma2(acc[i][j][0], kk, z0);
                            c_ffma2(acc[i][j][1], kk, z1);
                            c_ffma2(acc[i][j][2], kk, z2);
                            c_ffma2(acc[i][j][3], kk, z3);
                        }
                    hh = hn;
                    geo = geon;
                }
            };

            // the first n entries of the hit list, in batches: A2 | sync | B | sync
            auto process_list = [&](int n) {
                for (int b0 = 0; b0 < n; b0 += kcBatch) {
                    const int nbat = min(kcBatch, n - b0);
                    phase_a2(b0, nbat);
                    __syncthreads();
                    phase_b(nbat);
                    __syncthreads();
                }
            };

            // ---- scale range of the group and the bucket window it implies at the reference scale
            double s_lo = sc, s_hi = sc;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                s_lo = fmin(s_lo, __shfl_xor_sync(full, s_lo, o));
                s_hi = fmax(s_hi, __shfl_xor_sync(full, s_hi, o));
            }
            const double halfN = (double)(N / 2);
            const double cx0 = (double)X0 - halfN, cx1 = (double)(X0 + kcTileX - 1) - halfN;
            const double cy0 = (double)Y0 - halfN, cy1 = (double)(Y0 + kcTileY - 1) - halfN;
            int wx0 = 0, wx1 = P.nb - 1, wy0 = 0, wy1 = P.nb - 1;
            {
                const double s_ref = *P.scale_ref;
                const double rl = s_lo / s_ref, rh = s_hi / s_ref;
                if (rl > 1e-3 && rh <= 1.0 + 1e-9) {
                    const double pad = (double)hW + 1.25, il = 1.0 / rl, ih = 1.0 / rh;
                    const double ax = cx0 - pad, bxx = cx1 + pad, ay = cy0 - pad, byy = cy1 + pad;
                    const double ib = 1.0 / kBucketCells, top = (double)(P.nb - 1);
                    wx0 = (int)fmin(fmax(floor((fmin(ax * il, ax * ih) + halfN) * ib), 0.0), top);
                    wx1 = (int)fmin(fmax(floor((fmax(bxx * il, bxx * ih) + halfN) * ib), 0.0), top);
                    wy0 = (int)fmin(fmax(floor((fmin(ay * il, ay * ih) + halfN) * ib), 0.0), top);
                    wy1 = (int)fmin(fmax(floor((fmax(byy * il, byy * ih) + halfN) * ib), 0.0), top);
                }
            }

            // ---- A1: candidate rows -> hit list (flushed through A2 + B whenever it would overflow)
            int n_local = 0, n_total = 0, par = 0;
            for (int rg = wy0; rg <= wy1; rg += 32) {
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
                for (int base = 0; base < total; base += kcThreads) {
                    if (n_local + kcThreads > kcListCap) {                 // uniform: n_local is the same in all threads
                        __syncthreads();
                        process_list(n_local);
                        n_local = 0;
                    }
                    const int f = base + tid;
                    bool hit = false;
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
                    if (f < total) {
                        p = __ldg(P.uv_sorted + k);
                        const double xa = __dmul_rn(__dmul_rn(p.x, s_lo), P.g.inv_du), xb = __dmul_rn(__dmul_rn(p.x, s_hi), P.g.inv_du);
                        const double ya = __dmul_rn(__dmul_rn(p.y, s_lo), P.g.inv_du), yb = __dmul_rn(__dmul_rn(p.y, s_hi), P.g.inv_du);
                        hit = fmax(xa, xb) + P.reach >= cx0 && fmin(xa, xb) - P.reach <= cx1 &&
                              fmax(ya, yb) + P.reach >= cy0 && fmin(ya, yb) - P.reach <= cy1;
                    }
                    const unsigned ball = __ballot_sync(full, hit);
                    if (lane == 0) S.warp_cnt[par][warp] = __popc(ball);
                    __syncthreads();
                    int cv = lane < kcWarps ? S.warp_cnt[par][lane] : 0, ci = cv;
#pragma unroll
                    for (int o = 1; o < kcWarps; o <<= 1) {
                        const int t = __shfl_up_sync(full, ci, o);
                        if (lane >= o) ci += t;
                    }
                    const int tot = __shfl_sync(full, ci, kcWarps - 1);
                    const int wbase = __shfl_sync(full, ci - cv, warp);
                    if (hit) {
                        const int slot = n_local + wbase + __popc(ball & lt_mask);
                        S.hit_uv[slot] = p;
                        S.hit_row[slot] = __ldg(P.perm + k);
                    }
                    n_local += tot;
                    n_total += tot;
                    par ^= 1;
                }
            }
            __syncthreads();                                               // list complete; previous item's stage reads done
            process_list(n_local);

            // ---- a5: write the tile of all 32 channels and 4 pols, once
            if (n_total > 0) {
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
            {
                const int j = tid & 7, row = (tid >> 3) & 7, q0 = tid >> 6;      // 16 B chunk, tile row, (channel, pol) slot
                const int y = Y0 + row, x = X0 + 2 * j, pol = q0 & 3;
                if (y < N && x < N) {
                    const unsigned char* src = S.zs + (q0 >> 2) * kcChanStride + (pol * kcTileY + row) * 128 + j * 16;
                    float* dst = P.grid + (((size_t)(c0 + (q0 >> 2)) * 4 + pol) * plane + (size_t)y * N + x) * 2;
                    const int nch = min(kcLanes, P.n_chan - c0);
#pragma unroll 4
                    for (int ch = q0 >> 2; ch < nch; ch += 2) {
                        float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
                        if (n_total > 0) v = *reinterpret_cast<const float4*>(src);
                        c_st_stream_v4(dst, v);
                        src += 2 * kcChanStride;
                        dst += 2 * 4 * plane * 2;
                    }
                }
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
    P.scale_ref = p->ws.d_scale_ref;
    P.bucket_start = p->ws.d_bucket_count;
    P.perm = p->ws.d_perm;
    P.uv_sorted = p->ws.d_uv_sorted;
    P.tile_order = p->ws.d_tile_order;
    P.counter = p->ws.d_misc + 1;
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
    const long long n_items = (long long)P.nt * P.nt * 2 * P.n_groups;
    if (n_items >= 0x7fffffffLL) { set_error("design CHAN: too many work items"); return false; }
    P.n_items = (int)n_items;
    const size_t smem = chan_smem_bytes(P);
    auto kern = w ? chan_kernel<true> : chan_kernel<false>;
    static bool attr_set[2] = {false, false};
    if (!attr_set[w ? 1 : 0]) {
        if (!cuda_ok(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024), "chan smem attribute"))
            return false;
        attr_set[w ? 1 : 0] = true;
    }
    long long blocks = p->sm_count;
    if (blocks > n_items) blocks = n_items;
    if (blocks < 1) blocks = 1;
    kern<<<(unsigned)blocks, kcThreads, smem, st>>>(P);
    p->last_launches += 1;
    return cuda_ok(cudaGetLastError(), "chan_kernel");
}

}  // namespace mwa
