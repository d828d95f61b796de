// index.cuh - the one index function every kernel of the library uses.
//
// DESIGN.md readings R1-R4: uv in metres, s_c = nu_c / c, x = (u_m * s_c) * inv_du, then
//   ka = floor(|x| * O + 0.5) ; q = ka div O ; rem = ka mod O ; if rem > O/2: q += 1, rem -= O
//   i = N/2 + sgn * q ; r = sgn * rem + O/2 ; valid iff the whole W-wide stamp lies in [0, N).
// Every fp64 step is an explicitly rounded intrinsic so that nvcc can never contract a multiply-add
// into an FMA: the result must equal the CPU evaluation bit for bit (BASELINE.json north_star).
#pragma once
#include <cuda_runtime.h>

namespace mwa {

constexpr double kSpeedOfLight = 299792458.0;   // R2: SI definition, exact

struct GridGeom {
    int N;          // grid cells per side
    int W;          // kernel support (odd)
    int h;          // (W - 1) / 2
    int O;          // oversampling (even)
    int o_shift;    // log2(O) when O is a power of two, else -1 (the division below then takes the generic path)
    double inv_du;  // 1.0 / cell_du, computed once on the host in fp64
};

// a1: per-channel scale, IEEE round-to-nearest division.
__device__ __forceinline__ double channel_scale(double freq_hz) { return __ddiv_rn(freq_hz, kSpeedOfLight); }

// Position in cells relative to the grid centre: two RN multiplies in this order (R3).
__device__ __forceinline__ double cell_coord(double metres, double scale, double inv_du) {
    return __dmul_rn(__dmul_rn(metres, scale), inv_du);
}

// INDEX(x) of R4.  Returns false (and leaves i, r untouched) for a dropped coordinate.
__device__ __forceinline__ bool index_1d(double x, const GridGeom& g, int& i, int& r) {
    const double a = fabs(x);
    if (!(a < (double)(g.N / 2))) return false;              // also rejects NaN / Inf before the int cast
    const int sgn = (__double2hiint(x) < 0) ? -1 : 1;        // signbit, so -0.0 behaves like the CPU's signbit()
    const double shifted = __dadd_rn(__dmul_rn(a, (double)g.O), 0.5);
    const int ka = __double2int_rd(shifted);                 // floor; < N/2 * O + 1 <= 2^20, fits easily
    int q, rem;                                              // non-negative integer division ka = q * O + rem
    if (g.o_shift >= 0) { q = ka >> g.o_shift; rem = ka & (g.O - 1); }
    else { q = ka / g.O; rem = ka - q * g.O; }
    if (rem > g.O / 2) { q += 1; rem -= g.O; }
    const int ii = g.N / 2 + sgn * q;
    if (ii - g.h < 0 || ii + g.h > g.N - 1) return false;    // R11: whole stamp must be inside
    i = ii;
    r = sgn * rem + g.O / 2;
    return true;
}

// The same INDEX(x) for a power-of-two O, written branch-free (K5's inner loop).  Identical results to index_1d:
//   |x| * O is exact for a power of two, so fma(|x|, O, 0.5) rounds once exactly like the multiply-then-add;
//   q' = (ka + O/2 - 1) >> log2 O carries exactly when rem > O/2;  rem' = ka - q' * O lies in [-O/2 + 1, O/2];
//   the sign is re-applied with the two's-complement identity (v ^ m) - m, m = 0 or -1.
// `origin` receives i - h (the first cell of the stamp); valid iff 0 <= origin <= N - W.
__device__ __forceinline__ bool index_1d_pow2(double x, const GridGeom& g, int& origin, int& r) {
    const double a = fabs(x);
    const bool in = a < (double)(g.N / 2);                    // false for NaN / Inf
    const int m = __double2hiint(x) >> 31;                    // 0 or -1 (signbit)
    const int ka = __double2int_rd(__fma_rn(a, (double)g.O, 0.5));
    const int q = (ka + (g.O / 2 - 1)) >> g.o_shift;
    const int rem = ka - (q << g.o_shift);
    origin = g.N / 2 - g.h + ((q ^ m) - m);
    r = ((rem ^ m) - m) + g.O / 2;
    return in && (unsigned)origin <= (unsigned)(g.N - g.W);
}

struct SampleIndex { int iu, iv, ru, rv; };

__device__ __forceinline__ bool sample_index(double um, double vm, double scale, const GridGeom& g, SampleIndex& s) {
    const double x = cell_coord(um, scale, g.inv_du);
    const double y = cell_coord(vm, scale, g.inv_du);
    if (g.o_shift >= 0) {                                     // uniform branch: every thread of a launch takes the same side
        int ou, ov, ru, rv;
        const bool oku = index_1d_pow2(x, g, ou, ru);
        const bool okv = index_1d_pow2(y, g, ov, rv);
        s.iu = ou + g.h; s.iv = ov + g.h; s.ru = ru; s.rv = rv;
        return oku && okv;
    }
    int iu, ru, iv, rv;
    const bool oku = index_1d(x, g, iu, ru);
    const bool okv = index_1d(y, g, iv, rv);
    if (!(oku && okv)) return false;
    s.iu = iu; s.iv = iv; s.ru = ru; s.rv = rv;
    return true;
}

}  // namespace mwa
