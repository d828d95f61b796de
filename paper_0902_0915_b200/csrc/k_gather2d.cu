// k_gather2d.cu - f3: gridding with a general 2-D COMPLEX kernel table ("general 2-D / complex
// kernel tables [O+1][O+1][W][W] (w-projection-style, 4 FMA per tap)"; PAPER.md:27 names only "a convolution"):
//
//     G[c][p][iv + tv - h][iu + tu - h] += K[rv][ru][tv][tu] * (w * V_p)              complex x complex, fp32 accumulate
//
// Same ownership as K3c (k_gather.cu): one warp owns a 16x16-cell tile of one channel, lane = 4x2-cell block with
// 8 cells x 4 pol x (re, im) = 64 fp32 accumulators in registers, no atomics, every cell written once (R10), bit-identical
// from run to run.  What differs: a tap is a complex number looked up per CELL in the 2-D table (it is not a product of
// two 1-D taps, so K3c's shifted zero-padded row copies do not apply): a lane reads the up to 8 taps of its block with
// predicated 8-byte loads straight from the table in global memory (31.8 KB at W = 7, O = 8: L1 / L2 resident) and spends
// 2 FFMA2 per cell and polarisation.  Phase A (lane = candidate, exact index, block mask) and the 32 x 32 bit transpose
// are K3c's; phase B is the plain per-lane list walk.  A variant for completeness of the ABI, measured but not tuned.
#include "plan.h"

namespace mwa {

constexpr int k2Warps = 4;
constexpr int k2Cap = 128;

struct Gather2dParams {
    GridGeom g;
    const double* scale;
    const double* scale_ref;
    const int* bucket_start;
    const int* perm;
    const double2* uv_sorted;
    const int* tile_order;
    int* counter;
    const float4* vis;
    const float* weights;
    const float2* table2d;      // [(O+1)][(O+1)][W][W] complex
    float* grid;
    int n_chan, nb, nt;
    long long n_items;
};

typedef unsigned long long u64;

__device__ __forceinline__ u64 g2_pack(float a, float b) {
    u64 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b));
    return r;
}
__device__ __forceinline__ void g2_unpack(u64 v, float& a, float& b) { asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v)); }
__device__ __forceinline__ void g2_ffma2(u64& d, u64 a, u64 b) { asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(d) : "l"(a), "l"(b)); }

__device__ __forceinline__ unsigned g2_transpose32(unsigned x, int lane) {
#pragma unroll
    for (int s = 0; s < 5; ++s) {
        const int j = 16 >> s;
        const unsigned m = s == 0 ? 0x0000FFFFu : s == 1 ? 0x00FF00FFu : s == 2 ? 0x0F0F0F0Fu : s == 3 ? 0x33333333u : 0x55555555u;
        const unsigned y = __shfl_xor_sync(0xffffffffu, x, j);
        x = (lane & j) ? ((x & ~m) | ((y >> j) & m)) : ((x & m) | ((y << j) & ~m));
    }
    return x;
}

struct Warp2dSmem {
    float4 z[k2Cap][2];      // w * V
    unsigned idx[k2Cap];     // (ou + 16) | (ov + 16) << 6 | ru << 12 | rv << 18 : stamp origin relative to the tile, table rows
    unsigned mask[k2Cap];
    int row[k2Cap];
};

__global__ void __launch_bounds__(k2Warps * 32)
gather2d_kernel(const Gather2dParams P) {
    __shared__ Warp2dSmem smem[k2Warps];
    const GridGeom g = P.g;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    Warp2dSmem* wsm = &smem[warp];
    const int bx = lane & 3, by = lane >> 2;
    const double s_ref = *P.scale_ref;
    const size_t plane = (size_t)g.N * g.N;
    const unsigned lt_mask = (1u << lane) - 1u;
    const int W = g.W, O1 = g.O + 1;

    long long item = 0;
    if (lane == 0) item = (long long)atomicAdd(P.counter, 1);
    item = __shfl_sync(0xffffffffu, item, 0);
    while (item < P.n_items) {
        long long next_item = 0;
        if (lane == 0) next_item = (long long)atomicAdd(P.counter, 1);
        const int trank = (int)(item / P.n_chan);
        const int c = (int)(item - (long long)trank * P.n_chan);
        const int tile = P.tile_order[trank];
        const int ty = tile / P.nt, tx = tile - ty * P.nt;
        const int X0 = tx * kTile, Y0 = ty * kTile;
        const double sc = P.scale[c];
        int bx0 = 0, bx1 = P.nb - 1, by0 = 0, by1 = P.nb - 1;
        {
            const double rho = sc / s_ref;
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
        u64 acc[2][4][4];
#pragma unroll
        for (int i = 0; i < 2; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j)
#pragma unroll
                for (int p = 0; p < 4; ++p) acc[i][j][p] = 0ull;
        int n_buf = 0;

        auto consume = [&](int n) {
            __syncwarp();
#pragma unroll
            for (int b = 0; b < k2Cap / 32; ++b) {                      // lane = hit: visibility + weight
                const int hidx = b * 32 + lane;
                if (hidx < n) {
                    const size_t sidx = (size_t)wsm->row[hidx] * P.n_chan + c;
                    const float4 va = __ldg(P.vis + 2 * sidx), vb = __ldg(P.vis + 2 * sidx + 1);
                    const float wt = P.weights ? __ldg(P.weights + sidx) : 1.0f;
                    wsm->z[hidx][0] = make_float4(wt * va.x, wt * va.y, wt * va.z, wt * va.w);
                    wsm->z[hidx][1] = make_float4(wt * vb.x, wt * vb.y, wt * vb.z, wt * vb.w);
                }
            }
            unsigned mw[k2Cap / 32];
#pragma unroll
            for (int b = 0; b < k2Cap / 32; ++b) {
                const int hidx = b * 32 + lane;
                const unsigned m = (hidx < n) ? wsm->mask[hidx] : 0u;
                mw[b] = (b * 32 < n) ? g2_transpose32(m, lane) : 0u;
            }
            __syncwarp();
#pragma unroll
            for (int b = 0; b < k2Cap / 32; ++b) {
                unsigned m = mw[b];
                while (__any_sync(0xffffffffu, m != 0u)) {
                    if (m != 0u) {
                        const int hidx = b * 32 + __ffs(m) - 1;
                        m &= m - 1u;
                        const unsigned id = wsm->idx[hidx];
                        const int ou = (int)(id & 63u) - 16, ov = (int)((id >> 6) & 63u) - 16;
                        const int ru = (int)((id >> 12) & 63u), rv = (int)((id >> 18) & 63u);
                        const float2* K = P.table2d + ((size_t)rv * O1 + ru) * W * W;
                        const float4 za = wsm->z[hidx][0], zb = wsm->z[hidx][1];
                        // z and its swapped pair per polarisation: (re, im) and (im, re)
                        const u64 z0 = g2_pack(za.x, za.y), z1 = g2_pack(za.z, za.w), z2 = g2_pack(zb.x, zb.y), z3 = g2_pack(zb.z, zb.w);
                        const u64 s0 = g2_pack(za.y, za.x), s1 = g2_pack(za.w, za.z), s2 = g2_pack(zb.y, zb.x), s3 = g2_pack(zb.w, zb.z);
#pragma unroll
                        for (int i = 0; i < 2; ++i) {
                            const int tv = 2 * by + i - ov;
#pragma unroll
                            for (int j = 0; j < 4; ++j) {
                                const int tu = 4 * bx + j - ou;
                                float2 k = make_float2(0.0f, 0.0f);
                                if ((unsigned)tv < (unsigned)W && (unsigned)tu < (unsigned)W) k = __ldg(K + tv * W + tu);
                                // (kr + i ki)(zr + i zi) = (kr zr - ki zi) + i (kr zi + ki zr)
                                const u64 kr = g2_pack(k.x, k.x), ki = g2_pack(-k.y, k.y);
                                g2_ffma2(acc[i][j][0], kr, z0); g2_ffma2(acc[i][j][0], ki, s0);
                                g2_ffma2(acc[i][j][1], kr, z1); g2_ffma2(acc[i][j][1], ki, s1);
                                g2_ffma2(acc[i][j][2], kr, z2); g2_ffma2(acc[i][j][2], ki, s2);
                                g2_ffma2(acc[i][j][3], kr, z3); g2_ffma2(acc[i][j][3], ki, s3);
                            }
                        }
                    }
                }
            }
            __syncwarp();
        };

        for (int byb = by0; byb <= by1; ++byb) {
            const int k0 = __ldg(P.bucket_start + byb * P.nb + bx0);
            const int k1 = __ldg(P.bucket_start + byb * P.nb + bx1 + 1);
            for (int kb = k0; kb < k1; kb += 32) {
                const int k = kb + lane;
                bool hit = false;
                unsigned id = 0, mask = 0;
                int row = 0;
                if (k < k1) {
                    const double2 p = __ldg(P.uv_sorted + k);
                    SampleIndex s;
                    if (sample_index(p.x, p.y, sc, g, s)) {
                        const int ou = s.iu - g.h - X0, ov = s.iv - g.h - Y0;
                        if (ou > -W && ou < kTile && ov > -W && ov < kTile) {
                            hit = true;
                            row = __ldg(P.perm + k);
                            id = (unsigned)(ou + 16) | ((unsigned)(ov + 16) << 6) | ((unsigned)s.ru << 12) | ((unsigned)s.rv << 18);
                            const int bxl = max(0, ou >> 2), bxh = min(3, (ou + W - 1) >> 2);
                            const int byl = max(0, ov >> 1), byh = min(7, (ov + W - 1) >> 1);
                            const unsigned m4 = (2u << bxh) - (1u << bxl);
                            const unsigned rows = 0x11111111u & (0xFFFFFFFFu >> (28 - 4 * byh)) & (0xFFFFFFFFu << (4 * byl));
                            mask = rows * m4;
                        }
                    }
                }
                const unsigned ball = __ballot_sync(0xffffffffu, hit);
                const int cnt = __popc(ball);
                if (cnt == 0) continue;
                if (n_buf + cnt > k2Cap) { consume(n_buf); n_buf = 0; }
                if (hit) {
                    const int slot = n_buf + __popc(ball & lt_mask);
                    wsm->idx[slot] = id;
                    wsm->mask[slot] = mask;
                    wsm->row[slot] = row;
                }
                n_buf += cnt;
            }
        }
        if (n_buf > 0) consume(n_buf);

        const int x = X0 + 4 * bx;
        const bool v8 = (g.N & 3) == 0 && (reinterpret_cast<unsigned long long>(P.grid) & 31ull) == 0ull;
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            const int y = Y0 + 2 * by + i;
            if (y < g.N) {
#pragma unroll
                for (int p = 0; p < 4; ++p) {
                    float* dst = P.grid + (((size_t)c * 4 + p) * plane + (size_t)y * g.N + x) * 2;
                    float a0, a1, a2, a3;
                    if (v8) {                                    // one aligned 32-byte sector per lane: one 256-bit store (as K3c)
                        if (x < g.N) {
                            float a4, a5, a6, a7;
                            g2_unpack(acc[i][0][p], a0, a1);
                            g2_unpack(acc[i][1][p], a2, a3);
                            g2_unpack(acc[i][2][p], a4, a5);
                            g2_unpack(acc[i][3][p], a6, a7);
                            asm volatile("st.global.cs.v8.f32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"l"(dst), "f"(a0), "f"(a1), "f"(a2),
                                         "f"(a3), "f"(a4), "f"(a5), "f"(a6), "f"(a7) : "memory");
                        }
                        continue;
                    }
                    if (x + 1 < g.N) {
                        g2_unpack(acc[i][0][p], a0, a1);
                        g2_unpack(acc[i][1][p], a2, a3);
                        asm volatile("st.global.cs.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(dst), "f"(a0), "f"(a1), "f"(a2), "f"(a3) : "memory");
                    }
                    if (x + 3 < g.N) {
                        g2_unpack(acc[i][2][p], a0, a1);
                        g2_unpack(acc[i][3][p], a2, a3);
                        asm volatile("st.global.cs.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(dst + 4), "f"(a0), "f"(a1), "f"(a2), "f"(a3) : "memory");
                    }
                }
            }
        }
        item = __shfl_sync(0xffffffffu, next_item, 0);
    }
}

bool launch_gather2d(Plan* p, const float* vis, const float* w, long long n_vis, int n_chan, float* grid, cudaStream_t st) {
    (void)n_vis;
    if (p->geom.W > 15 || p->geom.O > 62) { set_error("2-D tables: W <= 15 and O <= 62"); return false; }
    Gather2dParams P;
    P.g = p->geom;
    P.scale = p->ws.d_scale;
    P.scale_ref = p->ws.d_scale_ref;
    P.bucket_start = p->ws.d_bucket_count;
    P.perm = p->ws.d_perm;
    P.uv_sorted = p->ws.d_uv_sorted;
    P.tile_order = p->ws.d_tile_order;
    P.counter = p->ws.d_misc;
    P.vis = (const float4*)vis;
    P.weights = w;
    P.table2d = (const float2*)p->d_table2d;
    P.grid = grid;
    P.n_chan = n_chan;
    P.nb = (p->geom.N + kBucketCells - 1) / kBucketCells;
    P.nt = (p->geom.N + kTile - 1) / kTile;
    P.n_items = (long long)P.nt * P.nt * n_chan;
    int ctas_per_sm = 0;
    if (!cuda_ok(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&ctas_per_sm, gather2d_kernel, k2Warps * 32, 0), "gather2d occupancy")) return false;
    if (ctas_per_sm < 1) ctas_per_sm = 1;
    long long want = (P.n_items + k2Warps - 1) / k2Warps;
    long long blocks = (long long)p->sm_count * ctas_per_sm;
    if (blocks > want) blocks = want;
    if (blocks < 1) blocks = 1;
    gather2d_kernel<<<(unsigned)blocks, k2Warps * 32, 0, st>>>(P);
    p->last_launches += 1;
    return cuda_ok(cudaGetLastError(), "gather2d_kernel");
}

}  // namespace mwa
