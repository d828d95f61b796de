// k_chan.cu - K5, the channel-SIMD register gridder (a2 + a4 + a5 fused) for finely channelised data.
//
// The correlator of PAPER.md:19 delivers 768 channels of 40 kHz: neighbouring channels see the same baseline
// at almost the same (u, v) (u_lambda = u_m * nu / c moves by 2.6e-4 of its radius per channel), and every
// channel owns its own grid (BASELINE.json configs[3]).  K5 turns that into SIMD lanes:
//
//   CTA  = one 16 x (4*passes) cell tile  x  one group of 32 adjacent channels (all 4 polarisations)
//   warp = one 4x2-cell block of the tile (8 warps cover 16x4 cells; `passes` sweeps cover the tile)
//   lane = one channel of the group; the lane keeps 8 cells x 4 pol x (re, im) = 64 fp32 accumulators
//          of ITS channel's grid in registers.
//
// All 32 lanes of a warp therefore walk (almost) the same list of baseline rows - the walk is balanced by
// construction, where K3c (k_gather.cu: lane = block, same channel) leaves 23 of 32 lanes idle on Poisson
// noise (profiles/r01_gather_v0_c4x64.md).  A lane whose stamp misses the block at its own channel reads
// zeros from the padded kernel table, so there is no divergence in the FMA body at all.
//
//   A1 (thread = candidate row): walk the uv buckets (k_bin.cu) that can reach the tile at ANY scale of the
//       channel group, keep the rows whose stamp can overlap the tile (conservative fp64 interval test).
//   A2 (warp = hit, lane = channel): the exact index function (index.cuh) per (row, channel); per lane a
//       packed pair of kernel-table offsets ("geo"), per hit a bit mask of the blocks any lane touches.
//   B  (warp = block, lane = channel): for every hit that touches the block: 2 x LDG.128 of the lane's
//       visibility (32 lanes = 1 KB contiguous), LDS.128 + LDS.64 of kernel taps, 10 FMUL, 32 FFMA2.
//   write-out: through a swizzled 16 KB shared-memory stage so that every global store is a full 128 B line
//       of one (channel, pol, row); each cell of grid_out is written exactly once, zeros included (R10).
//
// No atomics on grid data; no fp64 in phase B.  Visibilities are read straight from global memory (L1/L2
// serve the ~10 warps that visit the same row), kernel-table rows live in shared memory.
#include "plan.h"

namespace mwa {

constexpr int kcWarps = 8;
constexpr int kcThreads = kcWarps * 32;
constexpr int kcLanes = 32;            // channels per group
constexpr int kcTileX = 16;
constexpr int kcListCap = 1024;        // candidate hits kept per A1 sweep (row id + uv)
constexpr int kcGeoCap = 128;          // hits per A2/B batch (geo: 128 x 32 x 4 B = 16 KB)
constexpr int kcPadU = 20;             // zero padding (floats) in front of a u table row
constexpr int kcZeroFloats = 32;       // all-zero block behind each table (target of an invalid lane's geo)
constexpr int kcStageBytes = 32 * 4 * 128;   // 32 channels x 4 rows x 128 B

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
    int passes;                 // 1, 2 or 4: tile height = 4 * passes
    int rlu, rlv, padv;         // padded row lengths of the shifted table copies, v padding
    int n_tu, n_tv;             // floats in the u / v table copies (zero blocks excluded)
    long long n_items;
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
    unsigned geo[kcGeoCap * kcLanes];
    double2 hit_uv[kcListCap];
    int hit_row[kcListCap];
    unsigned hit_mask[kcGeoCap];
    __align__(16) unsigned char stage[kcStageBytes];
    int n_hits;
    int item_lo, item_hi;         // next work item (64-bit, split)
};

template <bool HAS_W>
__global__ void __launch_bounds__(kcThreads, 2)
chan_kernel(const ChanParams P) {
    if (P.dispatch != nullptr && *P.dispatch != P.dispatch_want) return;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    ChanSmem& S = *reinterpret_cast<ChanSmem*>(smem_raw);
    float* tu = reinterpret_cast<float*>(smem_raw + ((sizeof(ChanSmem) + 15) & ~size_t(15)));
    float* tv = tu + P.n_tu + kcZeroFloats;
    const GridGeom g = P.g;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    // ---- shifted, zero-padded kernel-table copies (once per CTA)
    //   tu[s][r][q] = Tp_u[r][q + s], Tp_u[r][kcPadU + t] = T[r][t]     s = 0..3  (LDS.128 alignment)
    //   tv[s][r][q] = Tp_v[r][q + s], Tp_v[r][padv   + t] = T[r][t]     s = 0..1  (LDS.64 alignment)
    for (int k = tid; k < P.n_tu + kcZeroFloats; k += kcThreads) {
        float v = 0.0f;
        if (k < P.n_tu) {
            const int q = k % P.rlu, r = (k / P.rlu) % (g.O + 1), s = k / (P.rlu * (g.O + 1));
            const int t = q + s - kcPadU;
            if (t >= 0 && t < g.W) v = P.table[r * g.W + t];
        }
        tu[k] = v;
    }
    for (int k = tid; k < P.n_tv + kcZeroFloats; k += kcThreads) {
        float v = 0.0f;
        if (k < P.n_tv) {
            const int q = k % P.rlv, r = (k / P.rlv) % (g.O + 1), s = k / (P.rlv * (g.O + 1));
            const int t = q + s - P.padv;
            if (t >= 0 && t < g.W) v = P.table[r * g.W + t];
        }
        tv[k] = v;
    }
    if (tid == 0) { S.n_hits = 0; S.item_lo = atomicAdd(P.counter, 1); }
    __syncthreads();

    const int bx = warp & 3, byl = warp >> 2;
    const int TH = 4 * P.passes, nsub = 4 / P.passes;
    const unsigned tu_s = (unsigned)__cvta_generic_to_shared(tu) + 16u * bx;
    const unsigned tv_s = (unsigned)__cvta_generic_to_shared(tv);
    const unsigned zero_geo = (unsigned)(P.n_tu * 4) | ((unsigned)(P.n_tv * 4) << 16);
    const double s_ref = *P.scale_ref;
    const size_t plane = (size_t)g.N * g.N;
    const unsigned lt_mask = (1u << lane) - 1u;
    const unsigned full = 0xffffffffu;

    int item = S.item_lo;
    while (item < P.n_items) {
        int next_item = 0;
        if (tid == 0) next_item = atomicAdd(P.counter, 1);           // latency hidden behind this item
        const int grp = item % P.n_groups;
        const int ts = item / P.n_groups;
        const int sub = ts % nsub, trank = ts / nsub;
        const int tile = P.tile_order[trank];
        const int ty = tile / P.nt, tx = tile - ty * P.nt;
        const int X0 = tx * kcTileX, Y0 = ty * 16 + sub * TH;
        const int c0 = grp * kcLanes;
        const bool cvalid = c0 + lane < P.n_chan;
        const int cc = cvalid ? c0 + lane : P.n_chan - 1;
        const double sc = P.scale[cc];
        if (Y0 < g.N) {
        // ---- scale range of the group and the bucket window it implies at the reference scale
        double s_lo = sc, s_hi = sc;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            s_lo = fmin(s_lo, __shfl_xor_sync(full, s_lo, o));
            s_hi = fmax(s_hi, __shfl_xor_sync(full, s_hi, o));
        }
        const double halfN = (double)(g.N / 2);
        const double cx0 = (double)X0 - halfN, cx1 = (double)(X0 + kcTileX - 1) - halfN;
        const double cy0 = (double)Y0 - halfN, cy1 = (double)(Y0 + TH - 1) - halfN;
        int wx0 = 0, wx1 = P.nb - 1, wy0 = 0, wy1 = P.nb - 1;
        {
            const double rl = s_lo / s_ref, rh = s_hi / s_ref;
            if (rl > 1e-3 && rh <= 1.0 + 1e-9) {
                const double pad = (double)g.h + 1.25, il = 1.0 / rl, ih = 1.0 / rh;
                const double ax = cx0 - pad, bxx = cx1 + pad, ay = cy0 - pad, byy = cy1 + pad;
                const double ib = 1.0 / kBucketCells, top = (double)(P.nb - 1);
                wx0 = (int)fmin(fmax(floor((fmin(ax * il, ax * ih) + halfN) * ib), 0.0), top);
                wx1 = (int)fmin(fmax(floor((fmax(bxx * il, bxx * ih) + halfN) * ib), 0.0), top);
                wy0 = (int)fmin(fmax(floor((fmin(ay * il, ay * ih) + halfN) * ib), 0.0), top);
                wy1 = (int)fmin(fmax(floor((fmax(byy * il, byy * ih) + halfN) * ib), 0.0), top);
            }
        }
        const double reach = (double)g.h + 1.0;      // |x - ic| <= 1/2 + 1/(2O) <= 0.75, plus the half stamp

        u64 acc[2][4][4];   // [row i][col j][pol] = (re, im) of the lane's channel

        // ---- A2: exact indices of hits [b0, b0 + n) of the list for the lane's channel -> geo + block masks
        auto phase_a2 = [&](int b0, int n) {
            for (int hh = warp; hh < n; hh += kcWarps) {
                const double2 p = S.hit_uv[b0 + hh];
                SampleIndex s;
                unsigned geo = zero_geo, mask = 0u;
                if (cvalid && sample_index(p.x, p.y, sc, g, s)) {
                    const int ou = s.iu - g.h - X0, ov = s.iv - g.h - Y0;          // stamp origin relative to the tile
                    if (ou > -g.W && ou < kcTileX && ov > -g.W && ov < TH) {
                        const int su = (kcPadU - ou) & 3, sv = (P.padv - ov) & 1;
                        const int offu = (su * (g.O + 1) + s.ru) * P.rlu + (kcPadU - ou - su);
                        const int offv = (sv * (g.O + 1) + s.rv) * P.rlv + (P.padv - ov - sv);
                        geo = (unsigned)(offu * 4) | ((unsigned)(offv * 4) << 16);
                        const int bxl = max(0, ou >> 2), bxh = min(3, (ou + g.W - 1) >> 2);
                        const int bl = max(0, ov >> 1), bh = min(2 * P.passes - 1, (ov + g.W - 1) >> 1);
                        const unsigned m4 = (2u << bxh) - (1u << bxl);
                        const unsigned rows = 0x11111111u & (0xFFFFFFFFu >> (28 - 4 * bh)) & (0xFFFFFFFFu << (4 * bl));
                        mask = rows * m4;
                    }
                }
                mask = __reduce_or_sync(full, mask);
                S.geo[hh * kcLanes + lane] = geo;
                if (lane == 0) S.hit_mask[hh] = mask;
            }
        };

        // ---- B: the warp's block (bx, by) against hits [b0, b0 + n); every lane computes, zeros where it misses
        auto phase_b = [&](int b0, int n, int by) {
            const unsigned bit = (unsigned)(by * 4 + bx);
            const unsigned tvb = tv_s + 8u * by;
            unsigned m0, m1, m2, m3;
            {
                const unsigned k0 = lane < n ? S.hit_mask[lane] : 0u;
                const unsigned k1 = 32 + lane < n ? S.hit_mask[32 + lane] : 0u;
                const unsigned k2 = 64 + lane < n ? S.hit_mask[64 + lane] : 0u;
                const unsigned k3 = 96 + lane < n ? S.hit_mask[96 + lane] : 0u;
                m0 = __ballot_sync(full, (k0 >> bit) & 1u);
                m1 = __ballot_sync(full, (k1 >> bit) & 1u);
                m2 = __ballot_sync(full, (k2 >> bit) & 1u);
                m3 = __ballot_sync(full, (k3 >> bit) & 1u);
            }
            int gi = 0;
            unsigned m = m0;
            auto next_hit = [&]() -> int {
                if (m == 0u) {
                    if (gi < 1 && m1) { gi = 1; m = m1; }
                    else if (gi < 2 && m2) { gi = 2; m = m2; }
                    else if (gi < 3 && m3) { gi = 3; m = m3; }
                }
                if (m == 0u) return -1;
                const int b = __ffs(m) - 1;
                m &= m - 1u;
                return gi * 32 + b;
            };
            unsigned geo = 0;
            float4 va = make_float4(0, 0, 0, 0), vb = va;
            float wt = 1.0f;
            auto issue = [&](int hh) {
                geo = S.geo[hh * kcLanes + lane];
                const size_t sidx = (size_t)S.hit_row[b0 + hh] * P.n_chan + cc;
                va = __ldg(P.vis + 2 * sidx);
                vb = __ldg(P.vis + 2 * sidx + 1);
                if (HAS_W) wt = __ldg(P.weights + sidx);
            };
            int hh = next_hit();
            if (hh >= 0) issue(hh);
            while (hh >= 0) {
                const unsigned cgeo = geo;
                const float4 ca = va, cb = vb;
                const float cw = wt;
                hh = next_hit();
                if (hh >= 0) issue(hh);                                   // next visit's loads fly during the FMAs
                float ku0, ku1, ku2, ku3, kv0, kv1;
                asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(ku0), "=f"(ku1), "=f"(ku2), "=f"(ku3) : "r"(tu_s + (cgeo & 0xffffu)));
                asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(kv0), "=f"(kv1) : "r"(tvb + (cgeo >> 16)));
                if (HAS_W) { kv0 *= cw; kv1 *= cw; }
                const u64 z0 = c_pack2(ca.x, ca.y), z1 = c_pack2(ca.z, ca.w), z2 = c_pack2(cb.x, cb.y), z3 = c_pack2(cb.z, cb.w);
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
            }
        };

        // ---- write-out of the 4 tile rows of one pass: registers -> swizzled stage -> full 128 B lines
        auto write_pass = [&](int pass, bool zeros) {
            const int yb = Y0 + 4 * pass;
#pragma unroll 1
            for (int pol = 0; pol < 4; ++pol) {
                if (!zeros) {
                    __syncthreads();                                       // stage free (previous pol copied out)
#pragma unroll
                    for (int i = 0; i < 2; ++i) {
                        float a0, a1, a2, a3, b0, b1, b2, b3;
                        // pol is a run-time index: select with a small switch so the accumulators stay in registers
                        u64 e0, e1, e2, e3;
                        switch (pol) {
                            case 0: e0 = acc[i][0][0]; e1 = acc[i][1][0]; e2 = acc[i][2][0]; e3 = acc[i][3][0]; break;
                            case 1: e0 = acc[i][0][1]; e1 = acc[i][1][1]; e2 = acc[i][2][1]; e3 = acc[i][3][1]; break;
                            case 2: e0 = acc[i][0][2]; e1 = acc[i][1][2]; e2 = acc[i][2][2]; e3 = acc[i][3][2]; break;
                            default: e0 = acc[i][0][3]; e1 = acc[i][1][3]; e2 = acc[i][2][3]; e3 = acc[i][3][3]; break;
                        }
                        c_unpack2(e0, a0, a1); c_unpack2(e1, a2, a3); c_unpack2(e2, b0, b1); c_unpack2(e3, b2, b3);
                        unsigned char* rowp = S.stage + (lane * 4 + 2 * byl + i) * 128;
                        *reinterpret_cast<float4*>(rowp + (((2 * bx) ^ (lane & 7)) << 4)) = make_float4(a0, a1, a2, a3);
                        *reinterpret_cast<float4*>(rowp + (((2 * bx + 1) ^ (lane & 7)) << 4)) = make_float4(b0, b1, b2, b3);
                    }
                    __syncthreads();
                }
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const int idx = tid + kcThreads * k;
                    const int R = idx >> 3, j = idx & 7, ch = R >> 2, y = yb + (R & 3), x = X0 + 2 * j;
                    if (c0 + ch < P.n_chan && y < g.N && x < g.N) {
                        float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
                        if (!zeros) v = *reinterpret_cast<const float4*>(S.stage + R * 128 + ((j ^ (ch & 7)) << 4));
                        c_st_stream_v4(P.grid + (((size_t)(c0 + ch) * 4 + pol) * plane + (size_t)y * g.N + x) * 2, v);
                    }
                }
            }
        };

        // ---- A1 sweep for one pass; hits are flushed through A2 + B whenever the list would overflow.
        // Returns the number of hits left in the list; `flushed` says whether the list is incomplete.
        bool list_complete = false;
        int n_list = 0;
        auto sweep = [&](int by) {
            int n_local = 0;
            bool flushed = false;
            if (tid == 0) S.n_hits = 0;
            __syncthreads();
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
                        for (int b0 = 0; b0 < n_local; b0 += kcGeoCap) {
                            const int n = min(kcGeoCap, n_local - b0);
                            phase_a2(b0, n);
                            __syncthreads();
                            phase_b(b0, n, by);
                            __syncthreads();
                        }
                        if (tid == 0) S.n_hits = 0;
                        n_local = 0;
                        flushed = true;
                        __syncthreads();
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
                        const double xa = __dmul_rn(__dmul_rn(p.x, s_lo), g.inv_du), xb = __dmul_rn(__dmul_rn(p.x, s_hi), g.inv_du);
                        const double ya = __dmul_rn(__dmul_rn(p.y, s_lo), g.inv_du), yb2 = __dmul_rn(__dmul_rn(p.y, s_hi), g.inv_du);
                        hit = fmax(xa, xb) + reach >= cx0 && fmin(xa, xb) - reach <= cx1 &&
                              fmax(ya, yb2) + reach >= cy0 && fmin(ya, yb2) - reach <= cy1;
                    }
                    const unsigned ball = __ballot_sync(full, hit);
                    if (ball) {
                        int slot = 0;
                        if (lane == 0) slot = atomicAdd(&S.n_hits, __popc(ball));
                        slot = __shfl_sync(full, slot, 0) + __popc(ball & lt_mask);
                        if (hit) {
                            S.hit_uv[slot] = p;
                            S.hit_row[slot] = __ldg(P.perm + k);
                        }
                    }
                    n_local += __syncthreads_count(hit);
                }
            }
            n_list = n_local;
            list_complete = !flushed;
        };

        auto apply_list = [&](int by, bool geo_ready) {
            for (int b0 = 0; b0 < n_list; b0 += kcGeoCap) {
                const int n = min(kcGeoCap, n_list - b0);
                if (!geo_ready) {
                    phase_a2(b0, n);
                    __syncthreads();
                }
                phase_b(b0, n, by);
                if (b0 + kcGeoCap < n_list) __syncthreads();               // geo is overwritten by the next batch
            }
        };

        bool all_zero = false;
        for (int pass = 0; pass < P.passes && !all_zero; ++pass) {
            if (Y0 + 4 * pass >= g.N) break;
            const int by = 2 * pass + byl;
#pragma unroll
            for (int i = 0; i < 2; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j)
#pragma unroll
                    for (int p = 0; p < 4; ++p) acc[i][j][p] = 0ull;
            if (pass == 0 || !list_complete) {
                sweep(by);
                if (pass == 0 && list_complete && n_list == 0) {            // nothing reaches this tile in this group
                    all_zero = true;
                    break;
                }
                apply_list(by, false);
            } else {
                if (n_list > kcGeoCap) __syncthreads();                     // every warp is done with the last batch's geo
                apply_list(by, n_list <= kcGeoCap);                         // a single batch's geo is still in place
            }
            write_pass(pass, false);
        }
        if (all_zero)
            for (int pass = 0; pass < P.passes; ++pass)
                if (Y0 + 4 * pass < g.N) write_pass(pass, true);
        }   // Y0 < N

        __syncthreads();
        if (tid == 0) S.item_lo = next_item;
        __syncthreads();
        item = S.item_lo;
    }
}

// Geometry of the padded table copies for a tile of height 4 * passes (see the kernel header).
static void chan_table_geometry(const GridGeom& g, int passes, ChanParams& P) {
    const int TH = 4 * passes;
    P.passes = passes;
    P.rlu = (g.W + 35 + 3) & ~3;              // kcPadU + (W - 1) + 12 + 4, rounded up to a multiple of 4
    P.padv = TH;
    P.rlv = 2 * TH + g.W + 1;                 // even because W is odd
    P.n_tu = 4 * (g.O + 1) * P.rlu;
    P.n_tv = 2 * (g.O + 1) * P.rlv;
}

static size_t chan_smem_bytes(const ChanParams& P) {
    return ((sizeof(ChanSmem) + 15) & ~size_t(15)) + (size_t)(P.n_tu + P.n_tv + 2 * kcZeroFloats) * sizeof(float);
}

bool chan_supported(const Plan* p, int n_chan) {
    if (n_chan < 1) return false;
    ChanParams P;
    chan_table_geometry(p->geom, p->chan_passes, P);
    if ((P.n_tu + kcZeroFloats) * 4 > 65535 || (P.n_tv + kcZeroFloats) * 4 > 65535) return false;   // geo packs 16-bit byte offsets
    return chan_smem_bytes(P) <= 200 * 1024;
}

bool launch_chan(Plan* p, const float* vis, const float* w, long long n_vis, int n_chan, float* grid,
                 const int* dispatch, cudaStream_t st) {
    (void)n_vis;
    if (!chan_supported(p, n_chan)) { set_error("design CHAN does not support this kernel table size"); return false; }
    ChanParams P;
    P.g = p->geom;
    chan_table_geometry(p->geom, p->chan_passes, P);
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
    P.n_items = (long long)P.nt * P.nt * (4 / P.passes) * P.n_groups;
    if (P.n_items >= 0x7fffffffLL) { set_error("design CHAN: too many work items"); return false; }
    const size_t smem = chan_smem_bytes(P);
    auto kern = w ? chan_kernel<true> : chan_kernel<false>;
    static bool attr_set[2] = {false, false};
    if (!attr_set[w ? 1 : 0]) {
        if (!cuda_ok(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024), "chan smem attribute"))
            return false;
        attr_set[w ? 1 : 0] = true;
    }
    int ctas_per_sm = 0;
    if (!cuda_ok(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&ctas_per_sm, kern, kcThreads, smem), "chan occupancy"))
        return false;
    if (ctas_per_sm < 1) { set_error("chan kernel does not fit on an SM"); return false; }
    long long blocks = (long long)p->sm_count * ctas_per_sm;
    if (blocks > P.n_items) blocks = P.n_items;
    if (blocks < 1) blocks = 1;
    kern<<<(unsigned)blocks, kcThreads, smem, st>>>(P);
    p->last_launches += 1;
    return cuda_ok(cudaGetLastError(), "chan_kernel");
}

}  // namespace mwa
