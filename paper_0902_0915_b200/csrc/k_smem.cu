// k_smem.cu - K3a, the first comparison design of BASELINE.json north_star: tile-owned SHARED-MEMORY accumulation.
//
// One CTA owns one 32x32-cell tile of one channel (4 polarisations: 32 KB of complex64 in shared memory).  The
// kernel table is staged into shared memory with cp.async; the CTA walks the tile-sorted rows (the uv buckets of
// k_bin.cu that can reach the tile), and every warp scatters one hit at a time: lane = tap (W*W taps in rounds of
// 32 lanes), 8 x red.shared.add.f32 per tap.  When the walk is over the tile is written to the grid once, with
// full-line stores, zeros included - so, like K3c / K5, there is no zero-fill pass and no global atomic.
//
// It is here to be measured, not to be used (AUTO never picks it): the ncu numbers in profiles/ show the
// shared-memory atomic unit as its bound (one ATOMS per fp32 component: 8 W^2 per sample), which is why the
// product designs keep their accumulators in registers instead.
#include "plan.h"

namespace mwa {

constexpr int ksTile = 32;
constexpr int ksWarps = 8;
constexpr int ksThreads = ksWarps * 32;
constexpr int ksCap = 256;                 // hits buffered per sweep chunk

struct SmemParams {
    GridGeom g;
    const double* scale;        // [n_chan]
    const double* scale_ref;    // [1]
    const int* bucket_start;    // [nb*nb + 1]
    const double4* row_sorted;  // [n_vis] (u, v, row id, 0)
    int* counter;
    const float4* vis;
    const float* weights;
    const float* table;
    float* grid;
    int n_chan, nb, nts;        // nts = tiles per side
    long long n_items;
};

struct SmemHit { int iu, iv, ru, rv, row; };

__global__ void __launch_bounds__(ksThreads)
smem_kernel(const SmemParams P) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float* tile = reinterpret_cast<float*>(smem_raw);                       // [4 pol][32][32][2]
    float* tab = tile + 4 * ksTile * ksTile * 2;                            // [(O+1)][W], padded to 16 B
    const int n_tab = (P.g.O + 1) * P.g.W;
    SmemHit* hits = reinterpret_cast<SmemHit*>(tab + ((n_tab + 3) & ~3));
    __shared__ int s_item, s_nhits;
    const GridGeom g = P.g;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    // kernel table -> shared memory with cp.async (4 B granules: the table has no alignment guarantee beyond 4 B)
    for (int k = tid; k < n_tab; k += ksThreads)
        asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"((unsigned)__cvta_generic_to_shared(tab + k)), "l"(P.table + k) : "memory");
    asm volatile("cp.async.commit_group;" ::: "memory");
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    if (tid == 0) s_item = (int)atomicAdd(P.counter, 1);
    __syncthreads();

    const double s_ref = *P.scale_ref;
    const size_t plane = (size_t)g.N * g.N;
    const int WW = g.W * g.W;
    long long item = s_item;
    while (item < P.n_items) {
        const int c = (int)(item % P.n_chan);
        const int t = (int)(item / P.n_chan);
        const int ty = t / P.nts, tx = t - ty * P.nts;
        const int X0 = tx * ksTile, Y0 = ty * ksTile;
        const double sc = P.scale[c];
        for (int k = tid; k < 4 * ksTile * ksTile * 2; k += ksThreads) tile[k] = 0.0f;
        if (tid == 0) s_nhits = 0;
        __syncthreads();

        // bucket window of the tile (+ stamp halo) back-projected to the reference scale
        int bx0 = 0, bx1 = P.nb - 1, by0 = 0, by1 = P.nb - 1;
        {
            const double rho = sc / s_ref;
            if (rho > 1e-3 && rho <= 1.0 + 1e-9) {
                const double half = (double)(g.N / 2), pad = (double)g.h + 1.25, inv = 1.0 / rho, ib = 1.0 / kBucketCells, top = (double)(P.nb - 1);
                bx0 = (int)fmin(fmax(floor((((double)X0 - pad - half) * inv + half) * ib), 0.0), top);
                bx1 = (int)fmin(fmax(floor((((double)(X0 + ksTile - 1) + pad - half) * inv + half) * ib), 0.0), top);
                by0 = (int)fmin(fmax(floor((((double)Y0 - pad - half) * inv + half) * ib), 0.0), top);
                by1 = (int)fmin(fmax(floor((((double)(Y0 + ksTile - 1) + pad - half) * inv + half) * ib), 0.0), top);
            }
        }
        // scatter the buffered hits: warp = hit, lane = tap
        auto scatter = [&](int n) {
            for (int hh = warp; hh < n; hh += ksWarps) {
                const SmemHit h = hits[hh];
                const size_t sidx = (size_t)h.row * P.n_chan + c;
                const float4 va = __ldg(P.vis + 2 * sidx), vb = __ldg(P.vis + 2 * sidx + 1);
                const float wt = P.weights ? __ldg(P.weights + sidx) : 1.0f;
                const float z[8] = {wt * va.x, wt * va.y, wt * va.z, wt * va.w, wt * vb.x, wt * vb.y, wt * vb.z, wt * vb.w};
                for (int tap = lane; tap < WW; tap += 32) {
                    const int tv = tap / g.W, tu = tap - tv * g.W;
                    const int x = h.iu - g.h + tu - X0, y = h.iv - g.h + tv - Y0;
                    if (x >= 0 && x < ksTile && y >= 0 && y < ksTile) {
                        const float k = tab[h.rv * g.W + tv] * tab[h.ru * g.W + tu];
                        float* cell = tile + (y * ksTile + x) * 2;
#pragma unroll
                        for (int p = 0; p < 4; ++p) {
                            const unsigned a = (unsigned)__cvta_generic_to_shared(cell + p * ksTile * ksTile * 2);
                            asm volatile("red.shared.add.f32 [%0], %1;" ::"r"(a), "f"(k * z[2 * p]) : "memory");
                            asm volatile("red.shared.add.f32 [%0], %1;" ::"r"(a + 4u), "f"(k * z[2 * p + 1]) : "memory");
                        }
                    }
                }
            }
        };
        for (int byb = by0; byb <= by1; ++byb) {
            const int k0 = P.bucket_start[byb * P.nb + bx0], k1 = P.bucket_start[byb * P.nb + bx1 + 1];
            for (int kb = k0; kb < k1; kb += ksThreads) {
                const int k = kb + tid;
                bool hit = false;
                SmemHit h;
                if (k < k1) {
                    const double4 rec = P.row_sorted[k];
                    SampleIndex s;
                    if (sample_index(rec.x, rec.y, sc, g, s)) {
                        const int ou = s.iu - g.h - X0, ov = s.iv - g.h - Y0;
                        if (ou > -g.W && ou < ksTile && ov > -g.W && ov < ksTile) {
                            hit = true;
                            h.iu = s.iu; h.iv = s.iv; h.ru = s.ru; h.rv = s.rv; h.row = (int)rec.z;
                        }
                    }
                }
                // the buffer holds ksCap = ksThreads hits: scatter what is there before it could overflow
                if (__syncthreads_or(s_nhits + ksThreads > ksCap && s_nhits > 0)) {
                    scatter(s_nhits);
                    __syncthreads();
                    if (tid == 0) s_nhits = 0;
                    __syncthreads();
                }
                if (hit) hits[atomicAdd(&s_nhits, 1)] = h;
            }
        }
        __syncthreads();
        scatter(s_nhits);
        __syncthreads();

        // write-out: every cell of the tile once, 16 B per thread, full 128 B lines per quarter-warp
        for (int k = tid; k < 4 * ksTile * ksTile / 2; k += ksThreads) {        // float4 = 2 cells
            const int p = k / (ksTile * ksTile / 2), r = k - p * (ksTile * ksTile / 2);
            const int y = r / (ksTile / 2), x2 = r - y * (ksTile / 2);
            const int gy = Y0 + y, gx = X0 + 2 * x2;
            if (gy < g.N && gx < g.N) {
                const float4 v = *reinterpret_cast<const float4*>(tile + ((p * ksTile + y) * ksTile + 2 * x2) * 2);
                float* dst = P.grid + (((size_t)c * 4 + p) * plane + (size_t)gy * g.N + gx) * 2;
                asm volatile("st.global.cs.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(dst), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
            }
        }
        __syncthreads();
        if (tid == 0) s_item = (int)atomicAdd(P.counter, 1);
        __syncthreads();
        item = s_item;
    }
}

bool launch_smem(Plan* p, const float* vis, const float* w, long long n_vis, int n_chan, float* grid, cudaStream_t st) {
    (void)n_vis;
    SmemParams P;
    P.g = p->geom;
    P.scale = p->ws.d_scale;
    P.scale_ref = p->ws.d_scale_ref;
    P.bucket_start = p->ws.d_bucket_count;
    P.row_sorted = (const double4*)p->ws.d_row_sorted;
    P.counter = p->ws.d_misc + 2;
    P.vis = (const float4*)vis;
    P.weights = w;
    P.table = p->d_table;
    P.grid = grid;
    P.n_chan = n_chan;
    P.nb = (p->geom.N + kBucketCells - 1) / kBucketCells;
    P.nts = (p->geom.N + ksTile - 1) / ksTile;
    P.n_items = (long long)P.nts * P.nts * n_chan;
    if (P.n_items >= 0x7fffffffLL) { set_error("design SMEM: too many work items"); return false; }
    const int n_tab = (p->geom.O + 1) * p->geom.W;
    const size_t smem = (size_t)4 * ksTile * ksTile * 2 * 4 + (size_t)((n_tab + 3) & ~3) * 4 + sizeof(SmemHit) * ksCap;
    // a per-device setting: set on every launch (cheap)
    if (!cuda_ok(cudaFuncSetAttribute(smem_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024), "smem attribute")) return false;
    int ctas_per_sm = 0;
    if (!cuda_ok(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&ctas_per_sm, smem_kernel, ksThreads, smem), "smem occupancy")) return false;
    if (ctas_per_sm < 1) { set_error("smem kernel does not fit on an SM"); return false; }
    long long blocks = (long long)p->sm_count * ctas_per_sm;
    if (blocks > P.n_items) blocks = P.n_items;
    smem_kernel<<<(unsigned)blocks, ksThreads, smem, st>>>(P);
    p->last_launches += 1;
    return cuda_ok(cudaGetLastError(), "smem_kernel");
}

}  // namespace mwa
