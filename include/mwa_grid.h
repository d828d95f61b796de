/* mwa_grid.h - C ABI of the B200 convolutional visibility gridder.
 *
 * The operation (section 2.1): "The data-set then undergoes a convolution that interpolates
 * the samples onto a regular grid to permit the operation of the Fast Fourier Transform".  The input is
 * the correlator output of PAPER.md:19 (section 2): ~130,000 baselines x 768 channels x 4 polarisations,
 * complex.  Everything the paper leaves open (kernel function, support, rounding, layout, edge policy)
 * is fixed by the readings R1-R16 of DESIGN.md; the formulas below restate them.
 *
 *   h = (W-1)/2, s_c = freqs[c] / 299792458.0, x = (u_m * s_c) * (1.0 / cell_du)      (fp64, RN, no FMA)
 *   (iu, ru) = INDEX(x), (iv, rv) = INDEX(y)                                          (R4)
 *   grid[c][p][iv+tv-h][iu+tu-h] += T[rv][tv] * T[ru][tu] * w[n][c] * V[n][c][p]      (fp32 accumulate)
 *
 * All entry points are plain C; no torch types.  Pointers are DEVICE pointers unless the name or the
 * comment says host.  Functions return 0 (MWA_GRID_OK) or a negative error code; the text of the last
 * error on the calling thread is available from mwa_grid_last_error().
 */
#ifndef MWA_GRID_H
#define MWA_GRID_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mwa_grid_plan mwa_grid_plan; /* opaque */

enum {
    MWA_GRID_OK = 0,
    MWA_GRID_ERR_INVALID = -1, /* NULL / misaligned pointer, bad size or parameter */
    MWA_GRID_ERR_NOMEM = -2,   /* workspace allocation failed */
    MWA_GRID_ERR_CUDA = -3     /* CUDA runtime error; text in mwa_grid_last_error() */
};

/* Gridding designs (BASELINE.json north_star asks for the comparison).
 * AUTO picks CHAN when the call has >= 8 channels and every group of 32 adjacent channels moves a baseline
 * by at most 6 cells at the grid edge (decided on the device from freqs), else GATHER.
 * All designs give the same indices and values within the fp32 tolerance. */
enum {
    MWA_GRID_DESIGN_AUTO = 0,
    MWA_GRID_DESIGN_ATOMIC = 1, /* K0: memset + one global red.add per tap (bring-up / ncu baseline)        */
    MWA_GRID_DESIGN_SMEM = 2,   /* K3a: tile-owned shared-memory accumulation (red.shared.add.f32)          */
    MWA_GRID_DESIGN_ROMEIN = 3, /* K3b: threads own cells modulo W, register-resident, flush on cell change */
    MWA_GRID_DESIGN_GATHER = 4, /* K3c: tile-owned, lane = 4x2 cell block of one channel, registers              */
    MWA_GRID_DESIGN_CHAN = 5,   /* K5: tile-owned, lane = channel (32 adjacent channels per warp), registers     */
    MWA_GRID_DESIGN_CHANWS = 6, /* K6: K5's ownership as a warp-specialised producer / consumer pipeline: exact-index
                                   pre-pass, TMA bulk loads, mbarrier hand-off, tensor-map TMA stores (k_chanws.cu) */
    MWA_GRID_DESIGN_ROMEIN_SORTED = 7 /* K3b walking the rows in the uv-bucket order of the binning step instead of the
                                   caller's: the comparison design with the spatial locality a3 can give it */
};

/* Create a plan (R5-R8 for the table).
 *   grid_n        N, cells per side; even, 16 <= N <= 16384, N >= 2*support_W
 *   cell_du       wavelengths per cell, finite and > 0; the plan stores inv_du = 1.0 / cell_du (fp64)
 *   support_W     W, odd, 1 <= W <= 15
 *   oversample_O  O, even, 2 <= O <= 64
 *   kernel_table  HOST pointer, (O+1)*W floats, row-major [ru][t]; T[ru][t] is the 1-D kernel at the distance
 *                 from cell (ic + t - h) to a sample at ic + (ru - O/2)/O.  Copied; the caller keeps ownership.
 * Returns NULL on failure.  A plan owns one workspace (grown on first use, then reused: no allocation inside
 * a warmed-up call) and must not be used by two host threads at once; different plans are independent. */
mwa_grid_plan* mwa_grid_plan_create(int grid_n, double cell_du, int support_W, int oversample_O,
                                    const float* kernel_table);

/* f3 - a plan with a general 2-D COMPLEX kernel table (w-projection-style kernels, 4 FMA per tap):
 *   grid[c][p][iv+tv-h][iu+tu-h] += K[rv][ru][tv][tu] * w[n][c] * V[n][c][p]          (complex * complex, fp32 accumulate)
 *   kernel_table_2d  HOST pointer, (O+1)*(O+1)*W*W*2 floats, [rv][ru][tv][tu] (re, im); copied.  oversample_O <= 62.
 * Index function, drop rule and all layouts are those of mwa_grid_plan_create / mwa_grid_visibilities.  Such a plan grids
 * with one tile-owned register kernel (csrc/k_gather2d.cu; designs AUTO / GATHER) and does not take accumulate-into, MFS,
 * the imaging calls or the weights grid (they are defined for separable tables).  Returns NULL on failure. */
mwa_grid_plan* mwa_grid_plan_create_2d(int grid_n, double cell_du, int support_W, int oversample_O,
                                       const float* kernel_table_2d);

/* Grid one visibility set (hot path: SURVEY.md section 8(a) rows a1-a5).
 *   uv_f64   [n_vis][2]            double, metres (u_m, v_m)                 16-byte aligned
 *   freqs    [n_chan]              double, Hz
 *   vis_c64  [n_vis][n_chan][4][2] float (re, im), polarisation fastest      32-byte aligned
 *   weights  [n_vis][n_chan]       float, or NULL = all ones                 4-byte aligned
 *   grid_out [n_chan][4][N][N][2]  float (re, im), row = v, column = u       16-byte aligned
 *            OVERWRITTEN entirely: every cell is written, zeros where no tap lands (R10).
 *   stream   cudaStream_t passed as void* (0 = legacy default stream)
 * Samples whose stamp would leave the grid are dropped whole (R11); that is not an error, and the visibilities and
 * weights of dropped samples may hold anything (NaN flags included): they never reach a sum.  The visibilities and
 * weights of all OTHER samples must be finite: a sample is accumulated into whole 4 x 2-cell register blocks with zero
 * taps outside its stamp, so a NaN or Inf there would spread to up to 7 cells beyond the stamp (zero the flagged
 * samples - weight 0 and visibility 0 - before the call).
 * n_chan == 0 is a no-op; n_vis == 0 zero-fills the grid.  Asynchronous: returns after enqueue; the caller's
 * arrays must stay valid until the stream reaches the end of the call. */
int mwa_grid_visibilities(mwa_grid_plan* plan, const double* uv_f64, const double* freqs,
                          const float* vis_c64, const float* weights, long long n_vis, int n_chan,
                          float* grid_out, void* stream);

/* The same call on HOST buffers (pinned memory gives full PCIe speed; pageable works; no alignment requirement):
 * copies the inputs to a device staging area owned by the plan, grids, copies the grid back, and synchronises before
 * returning.  Channels own their grids, so the call is pipelined over ~8 chunks of channels (multiples of 32): the
 * upload of chunk k+1 and the download of chunk k-1's grids run on two copy streams of the plan under the gridding of
 * chunk k on `stream` (C4: 498 ms against 579 ms unpipelined; the 25.8 GB download at PCIe speed is what remains).
 * Each chunk bins its rows at its own top frequency, so values agree with the device call within the fp32 tolerance,
 * not bit for bit.  Not available with accumulate-into.  Layouts as above.  The end-to-end entry point bench.py times. */
int mwa_grid_visibilities_host(mwa_grid_plan* plan, const double* uv_f64, const double* freqs,
                               const float* vis_c64, const float* weights, long long n_vis, int n_chan,
                               float* grid_out, void* stream);

/* The gridding call for callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses
 * that forbid cudaMalloc): no plan, and no cudaMalloc / cudaFree / allocating library routine inside, on any call.
 * It runs the GATHER design (K3c: scale, binning, tile-owned register gridder - the kernels of the plan path) with the
 * binning workspace in a static device array of the library (csrc/k_noalloc.cu: about 7.6 MB of every GPU that loads
 * the library, held until exit), which fixes the maximum sizes of a call: */
#define MWA_GRID_NOALLOC_MAX_VIS 131072    /* rows per call (C4's 130,816 baselines fit)          */
#define MWA_GRID_NOALLOC_MAX_CHAN 1024     /* channels per call                                   */
#define MWA_GRID_NOALLOC_MAX_GRID_N 2048   /* grid cells per side                                 */
/* A call beyond any of them returns MWA_GRID_ERR_INVALID with a message naming the limit; nothing is enqueued.
 *   grid_n, cell_du, support_W, oversample_O   as in mwa_grid_plan_create (and grid_n <= the limit above)
 *   kernel_table_dev  DEVICE pointer, (O+1)*W floats, row-major [ru][t] as in mwa_grid_plan_create; read by the
 *                     kernels, not copied: it is the caller's and must stay valid until the stream reaches the end of
 *                     the call
 *   all other arguments: layouts, alignment, drop rule, finite-input contract and asynchrony of mwa_grid_visibilities;
 *   grid_out is overwritten entirely.
 * Values: those of a plan with MWA_GRID_DESIGN_GATHER, bit for bit (same kernels, same order of summation).
 * The first call on a device resolves the array's device address (cudaGetSymbolAddress) and loads the kernels: make it
 * before any region that forbids such set-up.  ALL calls on a device share the one array, which keeps the contents of
 * the call before (each call clears what it needs zeroed): calls that overlap on the GPU - two streams without an
 * ordering between them, two host threads - race on it and give wrong grids; order them on one stream or with events.
 * The current device must be the one the pointers live on.  Errors: MWA_GRID_ERR_INVALID / MWA_GRID_ERR_CUDA. */
int mwa_grid_visibilities_noalloc(int grid_n, double cell_du, int support_W, int oversample_O,
                                  const float* kernel_table_dev, const double* uv_f64, const double* freqs,
                                  const float* vis_c64, const float* weights, long long n_vis, int n_chan,
                                  float* grid_out, void* stream);

/* Test hook for "indices bit-exact": runs the SAME __device__ index function the gridders use.
 *   out_idx [n_vis][n_chan][4] int32 = (iu, iv, ru, rv), or (-1,-1,-1,-1) for a dropped sample. */
int mwa_grid_compute_indices(mwa_grid_plan* plan, const double* uv_f64, const double* freqs,
                             long long n_vis, int n_chan, int* out_idx, void* stream);

/* Companion weights grid: wgrid_out[c][y][x] = sum over the samples of channel c of
 * T[rv][tv] * T[ru][tu] * w - the gridded sampling density (what imaging weights and the normalisation of a dirty image are
 * derived from); it equals the real part of the XX grid of unit visibilities.
 *   wgrid_out [n_chan][N][N] float, DEVICE, overwritten; weights [n_vis][n_chan] or NULL = ones; other arguments as in
 *   mwa_grid_visibilities.  A by-product, written in scatter form (memset + one red.global.add.f32 per tap).  Asynchronous. */
int mwa_grid_weights_grid(mwa_grid_plan* plan, const double* uv_f64, const double* freqs, const float* weights, long long n_vis,
                          int n_chan, float* wgrid_out, void* stream);

/* Dropped-sample counter: the number of (row, channel) samples mwa_grid_visibilities would
 * drop for these coordinates (R11: a tap outside the grid, |x| >= N/2, or a non-finite coordinate), counted with the same
 * index function.  out_count is a HOST pointer.  Synchronous (it reads the count back). */
int mwa_grid_count_dropped(mwa_grid_plan* plan, const double* uv_f64, const double* freqs, long long n_vis, int n_chan,
                           long long* out_count, void* stream);

/* f3 - accumulate-into (the gridded data are "readily aggregated in frequency and time"; SURVEY.md section
 * 8(f)-3).  When enabled, mwa_grid_visibilities ADDS the gridded samples to what grid_out holds instead of overwriting it
 * (R10 then does not apply: cells no tap reaches are left as they are), so successive time steps or row batches can be
 * gridded onto the same grids.  K6 writes with reduce-add tensor-map stores and skips its zero-fill, K3c reads, adds and
 * writes its own cells, K0 / K3b skip their memset; the designs SMEM and CHAN return MWA_GRID_ERR_INVALID.  One fp32
 * rounding is added per call and cell.  Takes effect at the next call. */
int mwa_grid_plan_set_accumulate(mwa_grid_plan* plan, int enabled);

/* f3 - multi-frequency synthesis onto one shared grid ("readily aggregated in frequency"; SURVEY.md section
 * 8(f)-3).  When enabled, the samples of ALL channels of a call are summed onto ONE set of grids: grid_out is
 * [4][N][N][2] floats (n_chan = 1 planes) = sum over c of the per-channel grids of the default mode, overwritten (or
 * added to, with accumulate-into).  Different channels now write the same cells, so ownership ends at the tile: K3c adds
 * its register tiles with red.global.add.v4.f32, K0 and K3b (register ownership with flush on cell change - the workload
 * that design is made for) reduce as they always do; summation order and hence the last bits vary from run to run.
 * Designs: AUTO (= GATHER), GATHER, ATOMIC, ROMEIN, ROMEIN_SORTED; others return MWA_GRID_ERR_INVALID.  Next call on. */
int mwa_grid_plan_set_mfs(mwa_grid_plan* plan, int enabled);

/* Select the gridding design (MWA_GRID_DESIGN_*).  Takes effect at the next call. */
int mwa_grid_plan_set_design(mwa_grid_plan* plan, int design);

/* The design the last gridding call on this plan actually ran (MWA_GRID_DESIGN_*).  For AUTO this reads the
 * device-side decision back and therefore synchronises with the device; negative on error. */
int mwa_grid_plan_last_design(mwa_grid_plan* plan);

/* When enabled, every mwa_grid_visibilities call records CUDA events around its stages on `stream`.
 * mwa_grid_plan_stage_ms then synchronises on them and writes up to `n` floats (milliseconds) of the LAST
 * call into host array `out_ms`: [0] scale+binning (a1, a3), [1] gridding kernel(s) incl. any zero-fill
 * (a2, a4, a5), [2] whole call.  Returns the number of values written, or a negative error code. */
int mwa_grid_plan_set_profiling(mwa_grid_plan* plan, int enabled);
int mwa_grid_plan_stage_ms(mwa_grid_plan* plan, float* out_ms, int n);

/* ---- measurement utilities (csrc/k_probe.cu): not part of the gridding path, used by bench.py and profiles/ only ----
 * Measures the FP32 FMA throughput of the device with a register-only loop (the second term of the roofline of
 * BASELINE.json north_star needs a measured denominator): out_tflops[0] = fma.rn.f32, out_tflops[1] = fma.rn.f32x2,
 * both in TFLOP/s (2 flop per FMA).  HOST pointer to 2 doubles.  Synchronous; takes a few milliseconds. */
int mwa_grid_probe_fp32(mwa_grid_plan* plan, double* out_tflops, void* stream);

/* Conflict-free red.shared.add.f32 rate of the whole device in lane-atomics per second (every lane its own bank): the
 * peak that K3a's shared-memory atomic throughput is compared with.  HOST pointer to 1 double.  Synchronous. */
int mwa_grid_probe_smem_atomics(mwa_grid_plan* plan, double* out_rate, void* stream);

/* Test / diagnostics query (synchronises with the device): counters the last K6 gridding call left behind, written
 * into HOST array `out` (up to 32 values): [0] pipeline error code (0 = none; non-zero means a bounded wait inside the
 * kernel expired and the grid is incomplete), [1] work items, [2] items at least one sample reaches, [3] staged batches
 * of up to 16 hits, [4] largest number of hits of one item, [5] items whose hit list did not fit the pre-pass pool and
 * were swept inside the gridding kernel, [6] work items K5 served through its dense-tile path; with n >= 32 also [31]
 * work items of heavy tiles that K3c gridded with the four warps of a CTA (calls with few items per warp).  Returns the
 * number of values written. */
int mwa_grid_plan_last_stats(mwa_grid_plan* plan, long long* out, int n);

/* Test / diagnostics: caps the pool that holds K6's per-item hit lists at `entries` list entries (0 = default sizing,
 * 12 per (row, channel group)).  Items whose list finds no room are swept inside the gridding kernel - the same result
 * by a slower path, which the tests reach this way.  Takes effect at the next call. */
int mwa_grid_plan_set_list_pool(mwa_grid_plan* plan, long long entries);

/* Number of kernel launches (memsets included) enqueued by the last gridding call on this plan. */
int mwa_grid_plan_last_launches(const mwa_grid_plan* plan);

/* f1 - the two steps after gridding (Table 1 rows "FFT" and "Convolution Correction"; the
 * grid exists "to permit the operation of the Fast Fourier Transform"): for every N x N plane
 *   image[q'][p'] = sum_{j,i} grid[j][i] exp(+2 pi i ((i - N/2) p + (j - N/2) q) / N) / (c^(p) c^(q)),  p = p' - N/2, q = q' - N/2
 *   c^(p) = (1/O) sum'_{k=-WO/2..WO/2} C(k/O) cos(2 pi (k/O) p / N)   (end terms halved; C(k/O) read from the plan's table)
 * i.e. the unnormalised inverse transform of the grid with both centres at [N/2][N/2], divided by the transform of the
 * gridding kernel ("convolution correction").  The correction falls to ~2e-4 (W = 7) at the image edge, so only the
 * inner part of the image is meaningful (SURVEY.md pin P5).
 *   grid   [n_planes][N][N][2] float (re, im), DEVICE, as written by mwa_grid_visibilities (n_planes = n_chan * 4)
 *   image  [n_planes][N][N][2] float (re, im), DEVICE; may be the same buffer as grid (in place), else must not overlap
 * The transform is a batched cuFFT call (library), the shifts, the sign and the division are one fused in-place kernel.
 * Asynchronous on `stream` except for the first call on a plan (it builds c^ and synchronises once).  Returns 0 or a
 * negative error code (MWA_GRID_ERR_CUDA with "cuFFT ... could not be loaded" if the library is missing). */
int mwa_image_from_grid(mwa_grid_plan* plan, const float* grid, float* image, long long n_planes, void* stream);

/* f2 - Stokes conversion ("the measured instrumental polarization is converted into a set of Stokes
 * parameters by the application of a 4x4 matrix transformation.  This matrix is a function of time and position on the sky
 * ... and must be calculated ... for each pixel"; Table 1 row "Stokes Conversion").  The paper gives no
 * formula for the matrix, so the caller supplies it (R18):
 *   stokes_out[c][k][q][p] = sum_{j=0..3} matrix[q][p][k][j] * image[c][j][q][p]          (complex, fp32)
 *   image      [n_chan][4][N][N][2] float, DEVICE: the 4 instrumental planes XX, XY, YX, YY of every channel
 *   matrix     [N][N][4][4][2]      float, DEVICE, 16-byte aligned: one 4 x 4 complex matrix per pixel, row k, column j,
 *              shared by all channels of the call
 *   stokes_out [n_chan][4][N][N][2] float, DEVICE: planes k = 0..3 (I, Q, U, V for a Stokes matrix); may be `image`
 * One kernel, 32 B read + 32 B written per pixel and channel (HBM-bound).  Asynchronous on `stream`. */
int mwa_image_stokes(mwa_grid_plan* plan, const float* image, const float* matrix, float* stokes_out, int n_chan, void* stream);

/* The correction function of the plan: out_corr[p'] = c^(p' - N/2) for p' = 0..min(n, N)-1, HOST array of doubles.
 * Returns the number of values written.  Synchronous. */
int mwa_image_correction(mwa_grid_plan* plan, double* out_corr, int n);

/* Free the table and the workspace.  NULL is a no-op. */
void mwa_grid_plan_destroy(mwa_grid_plan* plan);

/* Text of the last error raised on the calling thread ("" if none).  Never NULL. */
const char* mwa_grid_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* MWA_GRID_H */
