/* TEST INFRASTRUCTURE - the CPU oracle.  Not part of the product; the CUDA library never calls it.
 *
 * Plain fp64 convolutional gridder: the definition of the operation written out as loops.
 * Source: PAPER.md:27 (section 2.1) - "The data-set then undergoes a convolution that interpolates the
 * samples onto a regular grid to permit the operation of the Fast Fourier Transform" - made concrete by
 * BASELINE.json (north_star, configs) and the readings R1-R16 listed in DESIGN.md.  The loop below is
 * the CPU-style "scatter" form the paper says its CPU code used.
 *
 *   G[c][p][iv+tv-h][iu+tu-h] += T[rv][tv] * T[ru][tu] * w[n][c] * V[n][c][p]       (all in fp64)
 *   A[c][p][...]              += the same product with every factor replaced by its absolute value
 *
 * Shares no code with the CUDA path.  Build: gcc -O2 -ffp-contract=off -fno-fast-math -fopenmp.
 * Parity of this oracle against the paper's own gridder is UNPINNED (the paper prints no values);
 * it is pinned against the mathematics by tests/test_oracle_*.py (pins P1-P6 in DESIGN.md).
 */
#include <math.h>
#include <stdint.h>
#include <stddef.h>

#define ORACLE_C_LIGHT 299792458.0   /* R2: SI definition, exact */

/* INDEX(x) of DESIGN.md reading R4: round |x| to the nearest 1/O (half away from zero), split into
 * cell + sub-cell with the remainder kept in [-O/2, O/2], re-apply the sign (an exactly odd function).
 * Returns 1 and (i, r) if the whole W-wide stamp lies inside [0, N), else 0 (sample dropped, R11). */
int oracle_index(double x, int N, int W, int O, int *i_out, int *r_out)
{
    int h = (W - 1) / 2;
    *i_out = -1;
    *r_out = -1;
    if (!(fabs(x) < (double)(N / 2))) return 0;          /* also rejects NaN/Inf before the int cast */
    int sgn = signbit(x) ? -1 : 1;
    double a = fabs(x);
    double scaled = a * (double)O;                       /* RN multiply */
    double shifted = scaled + 0.5;                       /* RN add      */
    int64_t ka = (int64_t)floor(shifted);
    int64_t q = ka / O;
    int64_t rem = ka % O;
    if (rem > O / 2) { q += 1; rem -= O; }               /* rem in [-O/2+1, O/2] */
    int64_t ic = sgn * q;
    int64_t r = sgn * rem;                               /* r in [-O/2, O/2] */
    int64_t i = (int64_t)(N / 2) + ic;
    if (!(i - h >= 0 && i + h <= (int64_t)N - 1)) return 0;
    *i_out = (int)i;
    *r_out = (int)(r + O / 2);                           /* table row in [0, O] */
    return 1;
}

/* (iu, iv, ru, rv) of one sample, or all -1 if dropped.  R3: s = nu/c ; x = (u_m * s) * inv_du. */
static int sample_index(double um, double vm, double s, double inv_du, int N, int W, int O, int out[4])
{
    double x = (um * s) * inv_du;
    double y = (vm * s) * inv_du;
    int iu, ru, iv, rv;
    int oku = oracle_index(x, N, W, O, &iu, &ru);
    int okv = oracle_index(y, N, W, O, &iv, &rv);
    if (!(oku && okv)) { out[0] = out[1] = out[2] = out[3] = -1; return 0; }
    out[0] = iu; out[1] = iv; out[2] = ru; out[3] = rv;
    return 1;
}

/* out_idx [n_vis][n_chan][4] int32 */
void oracle_compute_indices(const double *uv, const double *freqs, long long n_vis, int n_chan,
                            int N, double cell_du, int W, int O, int *out_idx)
{
    double inv_du = 1.0 / cell_du;
    for (int c = 0; c < n_chan; ++c) {
        double s = freqs[c] / ORACLE_C_LIGHT;
        for (long long n = 0; n < n_vis; ++n)
            sample_index(uv[2 * n], uv[2 * n + 1], s, inv_du, N, W, O, out_idx + ((size_t)n * n_chan + c) * 4);
    }
}

/* uv [n_vis][2] f64 metres; freqs [n_chan] f64 Hz; vis [n_vis][n_chan][4][2] f32; weights [n_vis][n_chan]
 * f32 or NULL; table [(O+1)][W] f32.  G [n_chan][4][N][N][2] f64 and A [n_chan][4][N][N] f64 (A may be
 * NULL) are OVERWRITTEN (R10).  Channels own disjoint grids, so they are the only parallel axis.
 * Returns the number of threads used. */
int oracle_grid(const double *uv, const double *freqs, const float *vis, const float *weights,
                long long n_vis, int n_chan, int N, double cell_du, int W, int O, const float *table,
                double *G, double *A, int n_threads)
{
    int h = (W - 1) / 2;
    double inv_du = 1.0 / cell_du;
    size_t plane = (size_t)N * N;
    if (n_threads < 1) n_threads = 1;
    if (n_threads > n_chan) n_threads = n_chan > 0 ? n_chan : 1;
#pragma omp parallel for num_threads(n_threads) schedule(dynamic, 1)
    for (int c = 0; c < n_chan; ++c) {
        double *Gc = G + (size_t)c * 4 * plane * 2;
        double *Ac = A ? A + (size_t)c * 4 * plane : NULL;
        for (size_t k = 0; k < 4 * plane * 2; ++k) Gc[k] = 0.0;
        if (Ac) for (size_t k = 0; k < 4 * plane; ++k) Ac[k] = 0.0;
        double s = freqs[c] / ORACLE_C_LIGHT;
        for (long long n = 0; n < n_vis; ++n) {
            int id[4];
            if (!sample_index(uv[2 * n], uv[2 * n + 1], s, inv_du, N, W, O, id)) continue;
            int iu = id[0], iv = id[1], ru = id[2], rv = id[3];
            const float *v = vis + ((size_t)n * n_chan + c) * 8;
            double wt = weights ? (double)weights[(size_t)n * n_chan + c] : 1.0;
            double zre[4], zim[4], zabs[4];
            for (int p = 0; p < 4; ++p) {
                zre[p] = wt * (double)v[2 * p];
                zim[p] = wt * (double)v[2 * p + 1];
                zabs[p] = fabs(wt) * hypot((double)v[2 * p], (double)v[2 * p + 1]);
            }
            for (int tv = 0; tv < W; ++tv) {
                double kv = (double)table[rv * W + tv];
                size_t row = (size_t)(iv + tv - h) * N;
                for (int tu = 0; tu < W; ++tu) {
                    double k = kv * (double)table[ru * W + tu];
                    size_t cell = row + (size_t)(iu + tu - h);
                    for (int p = 0; p < 4; ++p) {
                        Gc[(p * plane + cell) * 2] += k * zre[p];
                        Gc[(p * plane + cell) * 2 + 1] += k * zim[p];
                        if (Ac) Ac[p * plane + cell] += fabs(k) * zabs[p];
                    }
                }
            }
        }
    }
    return n_threads;
}

/* The same gridder for a general 2-D COMPLEX kernel table ("general 2-D / complex kernel tables
 * [O+1][O+1][W][W] (w-projection-style, 4 FMA per tap)"):
 *     G[c][p][iv+tv-h][iu+tu-h] += K[rv][ru][tv][tu] * (w * V_p)          (complex * complex, fp64)
 *     A[c][p][..]               += |K[rv][ru][tv][tu]| * |w| * |V_p|
 * table2d [(O+1)][(O+1)][W][W][2] f32 (re, im), indexed [rv][ru][tv][tu]; everything else as oracle_grid (same index
 * function, same drop rule R11, same layouts).  A separable real table K = T[rv][tv] * T[ru][tu] gives oracle_grid. */
int oracle_grid_2d(const double *uv, const double *freqs, const float *vis, const float *weights,
                   long long n_vis, int n_chan, int N, double cell_du, int W, int O, const float *table2d,
                   double *G, double *A, int n_threads)
{
    int h = (W - 1) / 2, O1 = O + 1;
    double inv_du = 1.0 / cell_du;
    size_t plane = (size_t)N * N;
    if (n_threads < 1) n_threads = 1;
    if (n_threads > n_chan) n_threads = n_chan > 0 ? n_chan : 1;
#pragma omp parallel for num_threads(n_threads) schedule(dynamic, 1)
    for (int c = 0; c < n_chan; ++c) {
        double *Gc = G + (size_t)c * 4 * plane * 2;
        double *Ac = A ? A + (size_t)c * 4 * plane : NULL;
        for (size_t k = 0; k < 4 * plane * 2; ++k) Gc[k] = 0.0;
        if (Ac) for (size_t k = 0; k < 4 * plane; ++k) Ac[k] = 0.0;
        double s = freqs[c] / ORACLE_C_LIGHT;
        for (long long n = 0; n < n_vis; ++n) {
            int id[4];
            if (!sample_index(uv[2 * n], uv[2 * n + 1], s, inv_du, N, W, O, id)) continue;
            int iu = id[0], iv = id[1], ru = id[2], rv = id[3];
            const float *v = vis + ((size_t)n * n_chan + c) * 8;
            double wt = weights ? (double)weights[(size_t)n * n_chan + c] : 1.0;
            const float *K = table2d + (((size_t)rv * O1 + ru) * W * W) * 2;
            for (int tv = 0; tv < W; ++tv) {
                size_t row = (size_t)(iv + tv - h) * N;
                for (int tu = 0; tu < W; ++tu) {
                    double kr = (double)K[(tv * W + tu) * 2], ki = (double)K[(tv * W + tu) * 2 + 1];
                    size_t cell = row + (size_t)(iu + tu - h);
                    for (int p = 0; p < 4; ++p) {
                        double zr = wt * (double)v[2 * p], zi = wt * (double)v[2 * p + 1];
                        Gc[(p * plane + cell) * 2] += kr * zr - ki * zi;
                        Gc[(p * plane + cell) * 2 + 1] += kr * zi + ki * zr;
                        if (Ac) Ac[p * plane + cell] += hypot(kr, ki) * fabs(wt) * hypot((double)v[2 * p], (double)v[2 * p + 1]);
                    }
                }
            }
        }
    }
    return n_threads;
}
