// k_basic.cu - a1 (per-channel scale), the index test hook, and K0: the global-atomic gridder.
//
// K0 is the bring-up path and the ncu baseline of the design comparison: it pays the
// grid bytes twice (zero-fill + read-modify-write in L2) and one red.global per tap.  PAPER.md:49 explains
// why the 2008 design avoided exactly this ("lacks an atomic floating point accumulate"); sm_100a has the
// instruction, which makes the scatter form legal but still not fast.
#include "plan.h"
#include "scale.cuh"

namespace mwa {

__global__ void scale_kernel(const double* __restrict__ freqs, int n_chan, int half_n, int chan_ok,
                             double* __restrict__ scale, double* __restrict__ scale_ref, int* __restrict__ dispatch,
                             double4* __restrict__ group) {
    pdl_release();                                      // bin_count_kernel may follow as a programmatic dependent (it waits for this grid)
    scale_block(freqs, n_chan, half_n, chan_ok, scale, scale_ref, dispatch, group);     // one block
}

bool launch_scale(Plan* p, const double* freqs, int n_chan, cudaStream_t st) {
    scale_kernel<<<1, 256, 0, st>>>(freqs, n_chan, p->geom.N / 2, (chan_supported(p, n_chan) || chanws_supported(p, n_chan)) ? 1 : 0, p->ws.d_scale,
                                    p->ws.d_scale_ref, p->ws.d_dispatch, (double4*)p->ws.d_group);
    p->last_launches += 1;
    return cuda_ok(cudaGetLastError(), "scale_kernel");
}

// ---------------------------------------------------------------- index hook (K4)
__global__ void indices_kernel(GridGeom g, const double2* __restrict__ uv, const double* __restrict__ scale,
                               long long n_vis, int n_chan, int4* __restrict__ out) {
    const long long total = n_vis * (long long)n_chan;
    for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < total;
         k += (long long)gridDim.x * blockDim.x) {
        const long long n = k / n_chan;
        const int c = (int)(k - n * n_chan);
        const double2 p = uv[n];
        SampleIndex s;
        int4 o = make_int4(-1, -1, -1, -1);
        if (sample_index(p.x, p.y, scale[c], g, s)) o = make_int4(s.iu, s.iv, s.ru, s.rv);
        out[k] = o;
    }
}

// ---------------------------------------------------------------- companion weights grid
// wgrid[c][y][x] = sum over samples of T[rv][tv] T[ru][tu] w  - the gridded sampling density that imaging weights and the
// normalisation of a dirty image are derived from; equal to the real part of the XX grid of unit visibilities.  One thread
// per (sample, tap row), one red.global.add.f32 per tap (K0's scatter form: this grid is a by-product, not the hot path).
__global__ void weights_grid_kernel(GridGeom g, const double2* __restrict__ uv, const double* __restrict__ scale,
                                    const float* __restrict__ weights, const float* __restrict__ table, long long n_vis,
                                    int n_chan, float* __restrict__ wgrid) {
    const long long total = n_vis * (long long)n_chan * g.W;
    const size_t plane = (size_t)g.N * g.N;
    for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < total; k += (long long)gridDim.x * blockDim.x) {
        const long long sample = k / g.W;
        const int tv = (int)(k - sample * g.W);
        const long long n = sample / n_chan;
        const int c = (int)(sample - n * n_chan);
        const double2 p = uv[n];
        SampleIndex s;
        if (!sample_index(p.x, p.y, scale[c], g, s)) continue;
        const float wt = weights ? weights[sample] : 1.0f;
        const float kv = table[s.rv * g.W + tv] * wt;
        float* base = wgrid + (size_t)c * plane + (size_t)(s.iv + tv - g.h) * g.N + (size_t)(s.iu - g.h);
        for (int tu = 0; tu < g.W; ++tu) atomicAdd(base + tu, kv * table[s.ru * g.W + tu]);
    }
}

bool launch_weights_grid(Plan* p, const double* uv, const float* w, long long n_vis, int n_chan, float* wgrid, cudaStream_t st) {
    const size_t bytes = (size_t)n_chan * p->geom.N * p->geom.N * 4;
    if (!cuda_ok(cudaMemsetAsync(wgrid, 0, bytes, st), "memset weights grid")) return false;
    p->last_launches += 1;
    const long long total = n_vis * (long long)n_chan * p->geom.W;
    if (total == 0) return true;
    long long blocks = (total + 255) / 256;
    if (blocks > (long long)p->sm_count * 32) blocks = (long long)p->sm_count * 32;
    weights_grid_kernel<<<(unsigned)blocks, 256, 0, st>>>(p->geom, (const double2*)uv, p->ws.d_scale, w, p->d_table, n_vis, n_chan, wgrid);
    p->last_launches += 1;
    return cuda_ok(cudaGetLastError(), "weights_grid_kernel");
}

// ---------------------------------------------------------------- dropped-sample counter
__global__ void count_dropped_kernel(GridGeom g, const double2* __restrict__ uv, const double* __restrict__ scale, long long n_vis,
                                     int n_chan, unsigned long long* __restrict__ count) {
    const long long total = n_vis * (long long)n_chan;
    unsigned long long mine = 0;
    for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < total; k += (long long)gridDim.x * blockDim.x) {
        const long long n = k / n_chan;
        const int c = (int)(k - n * n_chan);
        const double2 p = uv[n];
        SampleIndex s;
        mine += sample_index(p.x, p.y, scale[c], g, s) ? 0 : 1;
    }
    mine = __reduce_add_sync(0xffffffffu, (unsigned)mine);               // < 2^32 per warp pass: a thread sees < 2^27 samples
    if ((threadIdx.x & 31) == 0 && mine) atomicAdd(count, mine);
}

bool launch_count_dropped(Plan* p, const double* uv, long long n_vis, int n_chan, unsigned long long* d_count, cudaStream_t st) {
    const long long total = n_vis * (long long)n_chan;
    long long blocks = (total + 255) / 256;
    if (blocks > (long long)p->sm_count * 64) blocks = (long long)p->sm_count * 64;
    if (blocks < 1) blocks = 1;
    count_dropped_kernel<<<(unsigned)blocks, 256, 0, st>>>(p->geom, (const double2*)uv, p->ws.d_scale, n_vis, n_chan, d_count);
    p->last_launches += 1;
    return cuda_ok(cudaGetLastError(), "count_dropped_kernel");
}

bool launch_indices(Plan* p, const double* uv, long long n_vis, int n_chan, int* out_idx, cudaStream_t st) {
    const long long total = n_vis * (long long)n_chan;
    if (total == 0) return true;
    long long blocks = (total + 255) / 256;
    if (blocks > (long long)p->sm_count * 64) blocks = (long long)p->sm_count * 64;
    indices_kernel<<<(unsigned)blocks, 256, 0, st>>>(p->geom, (const double2*)uv, p->ws.d_scale, n_vis, n_chan,
                                                     (int4*)out_idx);
    p->last_launches += 1;
    return cuda_ok(cudaGetLastError(), "indices_kernel");
}

// ---------------------------------------------------------------- K0: one thread per (row, channel, tap row)
__device__ __forceinline__ void red_add_v2(float* addr, float a, float b) {
    asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" ::"l"(addr), "f"(a), "f"(b) : "memory");
}

__global__ void atomic_grid_kernel(GridGeom g, const double2* __restrict__ uv, const double* __restrict__ scale,
                                   const float4* __restrict__ vis, const float* __restrict__ weights,
                                   const float* __restrict__ table, long long n_vis, int n_chan,
                                   float* __restrict__ grid, int mfs) {
    const long long total = n_vis * (long long)n_chan * g.W;
    const size_t plane = (size_t)g.N * g.N;
    for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < total;
         k += (long long)gridDim.x * blockDim.x) {
        const long long sample = k / g.W;
        const int tv = (int)(k - sample * g.W);
        const long long n = sample / n_chan;
        const int c = (int)(sample - n * n_chan);
        const double2 p = uv[n];
        SampleIndex s;
        if (!sample_index(p.x, p.y, scale[c], g, s)) continue;
        const float wt = weights ? weights[sample] : 1.0f;
        const float4 va = vis[2 * sample], vb = vis[2 * sample + 1];
        const float z[8] = {wt * va.x, wt * va.y, wt * va.z, wt * va.w, wt * vb.x, wt * vb.y, wt * vb.z, wt * vb.w};
        const float kv = table[s.rv * g.W + tv];
        float* base = grid + ((size_t)(mfs ? 0 : c) * 4 * plane + (size_t)(s.iv + tv - g.h) * g.N + (size_t)(s.iu - g.h)) * 2;
        for (int tu = 0; tu < g.W; ++tu) {
            const float kk = kv * table[s.ru * g.W + tu];
#pragma unroll
            for (int pol = 0; pol < 4; ++pol)
                red_add_v2(base + (pol * plane + tu) * 2, kk * z[2 * pol], kk * z[2 * pol + 1]);
        }
    }
}

bool launch_atomic(Plan* p, const double* uv, const float* vis, const float* w, long long n_vis, int n_chan,
                   float* grid, cudaStream_t st) {
    const size_t bytes = (size_t)(p->mfs ? 1 : n_chan) * 4 * p->geom.N * p->geom.N * 8;
    if (!p->accumulate) {                                       // accumulate-into: the atomics add onto what is there
        if (!cuda_ok(cudaMemsetAsync(grid, 0, bytes, st), "memset grid")) return false;
        p->last_launches += 1;
    }
    const long long total = n_vis * (long long)n_chan * p->geom.W;
    if (total == 0) return true;
    long long blocks = (total + 255) / 256;
    if (blocks > (long long)p->sm_count * 32) blocks = (long long)p->sm_count * 32;
    atomic_grid_kernel<<<(unsigned)blocks, 256, 0, st>>>(p->geom, (const double2*)uv, p->ws.d_scale,
                                                         (const float4*)vis, w, p->d_table, n_vis, n_chan, grid, p->mfs ? 1 : 0);
    p->last_launches += 1;
    return cuda_ok(cudaGetLastError(), "atomic_grid_kernel");
}

}  // namespace mwa
