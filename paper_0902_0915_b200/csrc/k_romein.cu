// k_romein.cu - K3b, the second comparison design of BASELINE.json north_star: register-resident per-thread
// grid-point ownership.  A CTA of W x W threads walks a chunk of rows of ONE channel in the order the caller
// gave them (baseline order); thread (a, b) owns the cells with (x mod W, y mod W) = (a, b), so the W x W stamp of
// any sample holds exactly one cell of every thread.  The thread keeps the running sum of its CURRENT cell in
// registers (4 pol x (re, im)) and only when the stamp moves on to another of its cells does it flush the sum
// with red.global.add - "no global atomics on the common path" when consecutive samples stay on the same cells.
// Each lane computes the index of one sample of a 32-row batch (coalesced uv / vis loads) and the batch is then
// replayed to all threads by warp shuffles.
//
// It is here to be measured (AUTO never picks it).  The design pays off when one grid receives long runs of
// neighbouring samples (time or frequency synthesis onto a shared grid).  In BASELINE.json's configs every
// channel owns its grid and consecutive rows of a channel are different baselines, so nearly every sample
// flushes: the ncu numbers in profiles/ show it bound by L2 atomics like K0, plus the zero-fill pass.
#include "plan.h"

namespace mwa {

constexpr int krChunk = 4096;              // rows per CTA

struct RomeinParams {
    GridGeom g;
    const double* scale;
    const double2* uv;          // [n_vis] caller order
    const int* perm;            // walk order: position -> row (the uv-bucket order of k_bin.cu), or null = caller order
    const float4* vis;
    const float* weights;
    const float* table;
    float* grid;
    long long n_vis;
    int n_chan, n_chunks;
    int mfs;                    // 1: every channel adds into the one shared grid [4][N][N] (multi-frequency synthesis)
};

__device__ __forceinline__ void rom_red_v2(float* addr, float a, float b) {
    asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" ::"l"(addr), "f"(a), "f"(b) : "memory");
}

__global__ void romein_kernel(const RomeinParams P) {
    extern __shared__ float tab[];                                   // [(O+1)][W]
    const GridGeom g = P.g;
    const int tid = threadIdx.x, lane = tid & 31;
    const int n_thr = g.W * g.W;
    for (int k = tid; k < (g.O + 1) * g.W; k += blockDim.x) tab[k] = P.table[k];
    __syncthreads();
    const int c = blockIdx.x % P.n_chan;
    const int chunk = blockIdx.x / P.n_chan;
    const long long r0 = (long long)chunk * krChunk, r1 = min(P.n_vis, r0 + krChunk);
    const double sc = P.scale[c];
    const bool owner = tid < n_thr;
    const int a = tid % g.W, b = tid / g.W;                          // owned residues (x mod W, y mod W)
    const size_t plane = (size_t)g.N * g.N;
    float acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    int cx = -1, cy = -1;                                            // the cell the sums belong to
    auto flush = [&]() {
        if (cx >= 0) {
            float* base = P.grid + ((size_t)(P.mfs ? 0 : c) * 4 * plane + (size_t)cy * g.N + cx) * 2;
#pragma unroll
            for (int p = 0; p < 4; ++p) rom_red_v2(base + p * plane * 2, acc[2 * p], acc[2 * p + 1]);
        }
    };
    for (long long rb = r0; rb < r1; rb += 32) {
        // lane = one sample of the batch
        const long long pos = rb + lane;
        int iu = -1, iv = 0, ru = 0, rv = 0;
        float z[8] = {0, 0, 0, 0, 0, 0, 0, 0};
        if (pos < r1) {
            const long long n = P.perm ? (long long)__ldg(P.perm + pos) : pos;
            const double2 p = P.uv[n];
            SampleIndex s;
            if (sample_index(p.x, p.y, sc, g, s)) {
                iu = s.iu; iv = s.iv; ru = s.ru; rv = s.rv;
                const size_t sidx = (size_t)n * P.n_chan + c;
                const float4 va = __ldg(P.vis + 2 * sidx), vb = __ldg(P.vis + 2 * sidx + 1);
                const float wt = P.weights ? __ldg(P.weights + sidx) : 1.0f;
                z[0] = wt * va.x; z[1] = wt * va.y; z[2] = wt * va.z; z[3] = wt * va.w;
                z[4] = wt * vb.x; z[5] = wt * vb.y; z[6] = wt * vb.z; z[7] = wt * vb.w;
            }
        }
        const int nb = (int)min(32LL, r1 - rb);
        for (int j = 0; j < nb; ++j) {
            const int siu = __shfl_sync(0xffffffffu, iu, j);
            if (siu < 0) continue;                                   // dropped sample (uniform across the warp)
            const int siv = __shfl_sync(0xffffffffu, iv, j), sru = __shfl_sync(0xffffffffu, ru, j), srv = __shfl_sync(0xffffffffu, rv, j);
            float sz[8];
#pragma unroll
            for (int q = 0; q < 8; ++q) sz[q] = __shfl_sync(0xffffffffu, z[q], j);
            if (owner) {
                // the one cell of the stamp [x0, x0 + W) x [y0, y0 + W) with this thread's residues
                const int x0 = siu - g.h, y0 = siv - g.h;
                int tu = (a - x0) % g.W; if (tu < 0) tu += g.W;
                int tv = (b - y0) % g.W; if (tv < 0) tv += g.W;
                const int x = x0 + tu, y = y0 + tv;
                if (x != cx || y != cy) {
                    flush();
                    cx = x; cy = y;
#pragma unroll
                    for (int q = 0; q < 8; ++q) acc[q] = 0.0f;
                }
                const float k = tab[srv * g.W + tv] * tab[sru * g.W + tu];
#pragma unroll
                for (int q = 0; q < 8; ++q) acc[q] = fmaf(k, sz[q], acc[q]);
            }
        }
    }
    if (owner) flush();
}

bool launch_romein(Plan* p, const double* uv, const float* vis, const float* w, long long n_vis, int n_chan, float* grid,
                   const int* perm, cudaStream_t st) {
    const size_t bytes = (size_t)(p->mfs ? 1 : n_chan) * 4 * p->geom.N * p->geom.N * 8;
    if (!p->accumulate) {                                       // accumulate-into: the reductions add onto what is there
        if (!cuda_ok(cudaMemsetAsync(grid, 0, bytes, st), "memset grid")) return false;
        p->last_launches += 1;
    }
    RomeinParams P;
    P.g = p->geom;
    P.scale = p->ws.d_scale;
    P.uv = (const double2*)uv;
    P.perm = perm;
    P.vis = (const float4*)vis;
    P.weights = w;
    P.table = p->d_table;
    P.grid = grid;
    P.n_vis = n_vis;
    P.n_chan = n_chan;
    P.mfs = p->mfs ? 1 : 0;
    P.n_chunks = (int)((n_vis + krChunk - 1) / krChunk);
    const long long blocks = (long long)P.n_chunks * n_chan;
    if (blocks == 0) return true;
    if (blocks >= 0x7fffffffLL) { set_error("design ROMEIN: too many blocks"); return false; }
    const int threads = ((p->geom.W * p->geom.W + 31) / 32) * 32;
    romein_kernel<<<(unsigned)blocks, threads, (size_t)(p->geom.O + 1) * p->geom.W * sizeof(float), st>>>(P);
    p->last_launches += 1;
    return cuda_ok(cudaGetLastError(), "romein_kernel");
}

}  // namespace mwa
