// scale.cuh - a1: the per-channel scale s_c = nu_c / c, the binning reference scale max s_c, the per-group scale ranges of
// K5 / K6 and the device-side choice of MWA_GRID_DESIGN_AUTO, as one block-wide routine shared by scale_kernel
// (k_basic.cu) and the fused pre-pass of small calls (k_bin.cu: bin_small_kernel).
#pragma once
#include "index.cuh"
#include "plan.h"

namespace mwa {

// The gridder for MWA_GRID_DESIGN_AUTO is picked on the device (the host never reads freqs): K5 / K6 need the 32
// channels of a group to see a baseline at almost the same cell.  drift = largest displacement, in cells at the grid
// edge, between the extreme channels of any group.
constexpr double kChanMaxDriftCells = 6.0;

// Run by ALL threads of ONE block (any size that is a multiple of 32, <= 1024).  Returns max |s_c| to every thread.
__device__ __forceinline__ double scale_block(const double* __restrict__ freqs, int n_chan, int half_n, int chan_ok,
                                              double* __restrict__ scale, double* __restrict__ scale_ref,
                                              int* __restrict__ dispatch, double4* __restrict__ group) {
    // one block; also reduces max(s_c) for the binning reference scale
    __shared__ double smax[32];
    __shared__ double sref;
    __shared__ int bad;
    if (threadIdx.x == 0) bad = 0;
    __syncthreads();
    double m = 0.0;
    for (int c = threadIdx.x; c < n_chan; c += blockDim.x) {
        const double s = channel_scale(freqs[c]);
        scale[c] = s;
        m = fmax(m, fabs(s));
    }
    for (int g0 = threadIdx.x * 32; g0 < n_chan; g0 += blockDim.x * 32) {      // one 32-channel group per thread
        double lo = channel_scale(freqs[g0]), hi = lo;
        for (int c = g0 + 1; c < min(n_chan, g0 + 32); ++c) {
            const double s = channel_scale(freqs[c]);
            lo = fmin(lo, s);
            hi = fmax(hi, s);
        }
        if (!(lo > 0.0) || !((hi - lo) / hi * (double)half_n <= kChanMaxDriftCells)) atomicOr(&bad, 1);
    }
    for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0) smax[threadIdx.x >> 5] = m;
    __syncthreads();
    if (threadIdx.x < 32) {
        m = (threadIdx.x < (blockDim.x >> 5)) ? smax[threadIdx.x] : 0.0;
        for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
        if (threadIdx.x == 0) {
            *scale_ref = m;
            sref = m;
            *dispatch = (chan_ok && n_chan >= kChanMinChannels && !bad) ? 1 : 0;
        }
    }
    __syncthreads();
    // per 32-channel group (K5): {s_lo, s_hi, s_ref / s_lo, s_ref / s_hi}; the last two are NaN when the group cannot
    // be back-projected to the reference scale (non-positive scales), which makes K5 scan every bucket
    for (int g0 = threadIdx.x * 32; g0 < n_chan; g0 += blockDim.x * 32) {
        double lo = channel_scale(freqs[g0]), hi = lo;
        for (int c = g0 + 1; c < min(n_chan, g0 + 32); ++c) {
            const double s = channel_scale(freqs[c]);
            lo = fmin(lo, s);
            hi = fmax(hi, s);
        }
        const double rl = lo / sref, rh = hi / sref;
        const bool ok = rl > 1e-3 && rh <= 1.0 + 1e-9;
        const double nan = __longlong_as_double(0x7ff8000000000000LL);
        group[g0 >> 5] = make_double4(lo, hi, ok ? 1.0 / rl : nan, ok ? 1.0 / rh : nan);
    }
    return sref;
}

}  // namespace mwa
