// k_image.cu - f1, the two steps that follow gridding in the paper's imaging pipeline (Table 1 rows
// "FFT" and "Convolution Correction"; the grid exists "to permit the operation of the Fast Fourier
// Transform"):
//
//   I[q][p] = sum_{j,i} G[j][i] exp(+2 pi i ((i - N/2) p + (j - N/2) q) / N) / (c^(p) c^(q)),     p, q in [-N/2, N/2)
//   c^(p)   = (1/O) sum'_{k = -WO/2}^{WO/2} C(k/O) cos(2 pi (k/O) p / N)        (end terms halved; SURVEY.md pin P5)
//
// with the samples C(k/O) of the gridding kernel read back from the plan's own table.  The transform itself is a plain
// batched 2-D complex FFT and is left to cuFFT (loaded with dlopen at the first imaging call, so the gridding path does
// not depend on it).  Neither shift is a pass over the data: with the grid centre at [N/2][N/2] and the image centre
// at [N/2][N/2], both for even N,
//
//   I[q'][p'] = (-1)^(p' + q') F[(q' + N/2) mod N][(p' + N/2) mod N] / (c^(p' - N/2) c^(q' - N/2)),   F = unnormalised
//   inverse DFT of the grid as it lies in memory,
//
// so ONE in-place kernel after the FFT swaps the quadrants, applies the checkerboard sign and divides by the
// correction: 8 B read + 8 B written per pixel, bound by HBM (C4: 51.5 GB -> 8.0 ms at 6454 GB/s).
#include <cufft.h>
#include <dlfcn.h>

#include "plan.h"

namespace mwa {

// ------------------------------------------------------------------------------------------------ cuFFT through dlopen
struct CufftApi {
    void* lib = nullptr;
    cufftResult (*PlanMany)(cufftHandle*, int, int*, int*, int, int, int*, int, int, cufftType, int) = nullptr;
    cufftResult (*SetStream)(cufftHandle, cudaStream_t) = nullptr;
    cufftResult (*ExecC2C)(cufftHandle, cufftComplex*, cufftComplex*, int) = nullptr;
    cufftResult (*Destroy)(cufftHandle) = nullptr;
    bool ok = false;
};

static CufftApi& cufft_api() {
    static CufftApi api;
    if (api.ok || api.lib) return api;
    const char* names[] = {"libcufft.so.11", "libcufft.so", "/usr/local/cuda/lib64/libcufft.so.11", "/usr/local/cuda/lib64/libcufft.so"};
    for (const char* n : names) {
        api.lib = dlopen(n, RTLD_NOW | RTLD_LOCAL);
        if (api.lib) break;
    }
    if (!api.lib) return api;
    api.PlanMany = reinterpret_cast<decltype(api.PlanMany)>(dlsym(api.lib, "cufftPlanMany"));
    api.SetStream = reinterpret_cast<decltype(api.SetStream)>(dlsym(api.lib, "cufftSetStream"));
    api.ExecC2C = reinterpret_cast<decltype(api.ExecC2C)>(dlsym(api.lib, "cufftExecC2C"));
    api.Destroy = reinterpret_cast<decltype(api.Destroy)>(dlsym(api.lib, "cufftDestroy"));
    api.ok = api.PlanMany && api.SetStream && api.ExecC2C && api.Destroy;
    return api;
}

void image_release(Plan* p) {
    CufftApi& api = cufft_api();
    for (int k = 0; k < 2; ++k)
        if (p->fft_batch[k] > 0 && api.ok) { api.Destroy((cufftHandle)p->fft_handle[k]); p->fft_batch[k] = 0; }
    if (p->d_inv_corr) { cudaFree(p->d_inv_corr); p->d_inv_corr = nullptr; }
    delete[] p->h_corr;
    p->h_corr = nullptr;
}

// ------------------------------------------------------------------------------------------------ correction function
// One thread per image coordinate p' (p = p' - N/2): the cosine sum in fp64.  The kernel sample C(k/O) sits in the table
// at tap m = round(k/O) (clamped to [-h, h]) of the row with sub-cell offset r = m O - k.
__global__ void correction_kernel(GridGeom g, const float* __restrict__ table, double* __restrict__ corr, float* __restrict__ inv_corr) {
    const int pp = blockIdx.x * blockDim.x + threadIdx.x;
    if (pp >= g.N) return;
    const int p = pp - g.N / 2, half = g.W * g.O / 2;
    double acc = 0.0;
    for (int k = -half; k <= half; ++k) {
        int m = (int)floor((double)k / (double)g.O + 0.5);
        m = min(max(m, -g.h), g.h);
        const int r = m * g.O - k;                                        // in [-O/2, O/2]
        const double c = (double)table[(r + g.O / 2) * g.W + (m + g.h)];
        const double wgt = (k == -half || k == half) ? 0.5 : 1.0;
        // the argument is reduced exactly in integers: cos(2 pi (k p mod N O) / (N O))
        const long long md = (long long)g.N * g.O;
        long long kp = ((long long)k * p) % md;
        if (kp < 0) kp += md;
        acc += wgt * c * cospi(2.0 * (double)kp / (double)md);
    }
    const double v = acc / (double)g.O;
    corr[pp] = v;
    inv_corr[pp] = (float)(1.0 / v);
}

// ------------------------------------------------------------------------------------------------ shift + sign + correction
// In place on F (the FFT output).  A thread takes two neighbouring pixels (p', p' + 1) of row q' < N/2 and their partners
// in row q' + N/2 at column (p' + N/2) mod N; N is even, so the pairs never straddle the half-row boundary.
__global__ void __launch_bounds__(256)
image_finish_kernel(float4* __restrict__ img, const float* __restrict__ inv_corr, int N, long long n_pairs_per_plane, long long total) {
    const long long stride = (long long)gridDim.x * blockDim.x;
    const int halfN = N / 2, pairs_per_row = N / 2;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += stride) {
        const long long plane = t / n_pairs_per_plane;
        const int rem = (int)(t - plane * n_pairs_per_plane);
        const int q = rem / pairs_per_row, pa = (rem - q * pairs_per_row) * 2;        // q < N/2, pa even
        const int pb = pa < halfN ? pa + halfN : pa - halfN;
        float4* base = img + plane * ((long long)N * N / 2);
        const long long ia = ((long long)q * N + pa) >> 1, ib = ((long long)(q + halfN) * N + pb) >> 1;
        const float4 fa = base[ia], fb = base[ib];
        const float sq = (q & 1) ? -1.0f : 1.0f;                                      // (-1)^(p' + q'), p' = pa even
        const float ca_q = inv_corr[q] * sq, cb_q = inv_corr[q + halfN] * ((halfN & 1) ? -sq : sq);
        const float ca0 = inv_corr[pa] * ca_q, ca1 = -inv_corr[pa + 1] * ca_q;        // pixel (q, pa), (q, pa + 1)
        const float pbs = (pb & 1) ? -1.0f : 1.0f;                                    // pb has the parity of N/2
        const float cb0 = inv_corr[pb] * cb_q * pbs, cb1 = -inv_corr[pb + 1] * cb_q * pbs;
        base[ia] = make_float4(fb.x * ca0, fb.y * ca0, fb.z * ca1, fb.w * ca1);
        base[ib] = make_float4(fa.x * cb0, fa.y * cb0, fa.z * cb1, fa.w * cb1);
    }
}

// The same for a grid whose half size is odd (N = 2 mod 4): one pixel pair per thread, scalar accesses.
__global__ void __launch_bounds__(256)
image_finish_generic_kernel(float2* __restrict__ img, const float* __restrict__ inv_corr, int N, long long n_pairs_per_plane, long long total) {
    const long long stride = (long long)gridDim.x * blockDim.x;
    const int halfN = N / 2;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += stride) {
        const long long plane = t / n_pairs_per_plane;
        const int rem = (int)(t - plane * n_pairs_per_plane);
        const int q = rem / N, pa = rem - q * N;
        const int pb = pa < halfN ? pa + halfN : pa - halfN;
        float2* base = img + plane * ((long long)N * N);
        const long long ia = (long long)q * N + pa, ib = (long long)(q + halfN) * N + pb;
        const float2 fa = base[ia], fb = base[ib];
        const float ca = inv_corr[pa] * inv_corr[q] * (((pa + q) & 1) ? -1.0f : 1.0f);
        const float cb = inv_corr[pb] * inv_corr[q + halfN] * (((pb + q + halfN) & 1) ? -1.0f : 1.0f);
        base[ia] = make_float2(fb.x * ca, fb.y * ca);
        base[ib] = make_float2(fa.x * cb, fa.y * cb);
    }
}

static bool ensure_correction(Plan* p, cudaStream_t st) {
    if (p->d_inv_corr) return true;
    const int N = p->geom.N;
    double* d_corr = nullptr;
    if (!cuda_ok(cudaMalloc((void**)&d_corr, (size_t)N * sizeof(double)), "cudaMalloc correction")) return false;
    if (!cuda_ok(cudaMalloc((void**)&p->d_inv_corr, (size_t)N * sizeof(float)), "cudaMalloc correction")) { cudaFree(d_corr); return false; }
    correction_kernel<<<(N + 127) / 128, 128, 0, st>>>(p->geom, p->d_table, d_corr, p->d_inv_corr);
    p->h_corr = new (std::nothrow) double[N];
    bool ok = p->h_corr && cuda_ok(cudaMemcpyAsync(p->h_corr, d_corr, (size_t)N * sizeof(double), cudaMemcpyDeviceToHost, st), "copy correction") &&
              cuda_ok(cudaStreamSynchronize(st), "correction_kernel");
    cudaFree(d_corr);
    if (!ok) { cudaFree(p->d_inv_corr); p->d_inv_corr = nullptr; delete[] p->h_corr; p->h_corr = nullptr; }
    return ok;
}

const double* image_correction_host(Plan* p, cudaStream_t st) { return ensure_correction(p, st) ? p->h_corr : nullptr; }

// cuFFT plans are cached for two batch sizes: the chunk and the remainder of the last call
static bool fft_handle(Plan* p, int batch, cufftHandle& h) {
    CufftApi& api = cufft_api();
    for (int k = 0; k < 2; ++k)
        if (p->fft_batch[k] == batch) { h = (cufftHandle)p->fft_handle[k]; return true; }
    const int slot = p->fft_batch[0] == 0 ? 0 : 1;
    if (p->fft_batch[slot] > 0) { api.Destroy((cufftHandle)p->fft_handle[slot]); p->fft_batch[slot] = 0; }
    int n[2] = {p->geom.N, p->geom.N};
    cufftHandle nh;
    const cufftResult r = api.PlanMany(&nh, 2, n, nullptr, 1, 0, nullptr, 1, 0, CUFFT_C2C, batch);
    if (r != CUFFT_SUCCESS) { set_error("cufftPlanMany failed (cufftResult " + std::to_string((int)r) + ")"); return false; }
    p->fft_handle[slot] = (int)nh;
    p->fft_batch[slot] = batch;
    h = nh;
    return true;
}

bool launch_image(Plan* p, const float* grid, float* image, long long n_planes, cudaStream_t st) {
    CufftApi& api = cufft_api();
    if (!api.ok) { set_error("cuFFT (libcufft.so.11) could not be loaded: the imaging step is unavailable"); return false; }
    if (!ensure_correction(p, st)) return false;
    const int N = p->geom.N;
    const long long plane_floats = (long long)N * N * 2;
    // planes per cuFFT call: bounded so that the plan's work area stays small next to the grid
    long long chunk = (256LL << 20) / (plane_floats * 4);
    if (chunk < 1) chunk = 1;
    if (chunk > n_planes) chunk = n_planes;
    for (long long p0 = 0; p0 < n_planes; p0 += chunk) {
        const int batch = (int)((n_planes - p0 < chunk) ? n_planes - p0 : chunk);
        cufftHandle h;
        if (!fft_handle(p, batch, h)) return false;
        if (api.SetStream(h, st) != CUFFT_SUCCESS) { set_error("cufftSetStream failed"); return false; }
        const cufftResult r = api.ExecC2C(h, (cufftComplex*)(grid + p0 * plane_floats), (cufftComplex*)(image + p0 * plane_floats), CUFFT_INVERSE);
        if (r != CUFFT_SUCCESS) { set_error("cufftExecC2C failed (cufftResult " + std::to_string((int)r) + ")"); return false; }
        const bool vec = (N % 4) == 0;
        const long long pairs_per_plane = vec ? (long long)(N / 2) * (N / 2) : (long long)(N / 2) * N, total = pairs_per_plane * batch;
        long long blocks = (total + 255) / 256;
        if (blocks > (long long)p->sm_count * 16) blocks = (long long)p->sm_count * 16;
        if (vec)
            image_finish_kernel<<<(unsigned)blocks, 256, 0, st>>>(reinterpret_cast<float4*>(image + p0 * plane_floats), p->d_inv_corr, N,
                                                                 pairs_per_plane, total);
        else
            image_finish_generic_kernel<<<(unsigned)blocks, 256, 0, st>>>(reinterpret_cast<float2*>(image + p0 * plane_floats),
                                                                         p->d_inv_corr, N, pairs_per_plane, total);
        p->last_launches += 2;
    }
    return cuda_ok(cudaGetLastError(), "image_finish_kernel");
}

}  // namespace mwa

// ------------------------------------------------------------------------------------------------ f2: Stokes conversion
// "the measured instrumental polarization is converted into a set of Stokes parameters by the application of a
// 4x4 matrix transformation.  This matrix is a function of time and position on the sky relative to the instrument and must
// be calculated by the RTS for each pixel" (Table 1 row "Stokes Conversion").  The paper gives no formula for
// the matrix, so it is an INPUT here (R18): one 4 x 4 complex matrix per pixel, shared by all channels of the
// call ("a function of time and position"), applied across the 4 polarisation planes of every channel:
//     out[c][k][q][p] = sum_j M[q][p][k][j] * image[c][j][q][p]
// One thread per pixel keeps its matrix in registers and walks a range of channels: 32 B read + 32 B written per pixel
// and channel (the 128 B matrix is read once per thread), bound by HBM.  In place is allowed (image == out).
namespace mwa {

__global__ void __launch_bounds__(256)
stokes_kernel(const float2* __restrict__ image, const float4* __restrict__ matrix, float2* __restrict__ out, int N, int n_chan,
              int chan_per_block) {
    const long long npix = (long long)N * N;
    const long long pix = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (pix >= npix) return;
    float2 m[4][4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const float4 a = __ldg(matrix + pix * 8 + k * 2), b = __ldg(matrix + pix * 8 + k * 2 + 1);
        m[k][0] = make_float2(a.x, a.y); m[k][1] = make_float2(a.z, a.w);
        m[k][2] = make_float2(b.x, b.y); m[k][3] = make_float2(b.z, b.w);
    }
    const int c0 = blockIdx.y * chan_per_block, c1 = min(n_chan, c0 + chan_per_block);
    for (int c = c0; c < c1; ++c) {
        const float2* src = image + (long long)c * 4 * npix + pix;
        float2 v[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) v[j] = src[(long long)j * npix];
        float2* dst = out + (long long)c * 4 * npix + pix;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            float re = 0.0f, im = 0.0f;
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                re = fmaf(m[k][j].x, v[j].x, re); re = fmaf(-m[k][j].y, v[j].y, re);
                im = fmaf(m[k][j].x, v[j].y, im); im = fmaf(m[k][j].y, v[j].x, im);
            }
            dst[(long long)k * npix] = make_float2(re, im);
        }
    }
}

bool launch_stokes(Plan* p, const float* image, const float* matrix, float* out, int n_chan, cudaStream_t st) {
    const int N = p->geom.N;
    const long long npix = (long long)N * N;
    const unsigned bx = (unsigned)((npix + 255) / 256);
    // enough blocks to fill the device even for a small image: split the channels over blockIdx.y
    int split = (int)(((long long)p->sm_count * 16 + bx - 1) / bx);
    if (split < 1) split = 1;
    if (split > n_chan) split = n_chan;
    const int per = (n_chan + split - 1) / split;
    dim3 grid(bx, (unsigned)((n_chan + per - 1) / per));
    stokes_kernel<<<grid, 256, 0, st>>>((const float2*)image, (const float4*)matrix, (float2*)out, N, n_chan, per);
    p->last_launches += 1;
    return cuda_ok(cudaGetLastError(), "stokes_kernel");
}

}  // namespace mwa
