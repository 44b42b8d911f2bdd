// rf_cutout.cu -- candidate cut-outs: the phased, dedispersed dynamic spectrum at a
// candidate pixel.  "those with S/N greater than a higher threshold ... have candidate visualizations
// made"; the visualisation shows "image and spectrum".  The image half
// is rf_debug_image (same kernels as the search); this file is the spectrum half.
//
// Reading A22: spec[r][ch] = (1/n_ch) sum_{kept bl} Re( s[bl][ch] e^{+2 pi i (iu x + iv y)/N} ), s = the
// dedispersed, dt-averaged Stokes-I visibility of output integration jj = t_idx - half_window + r (rows 8a-1,
// 8a-2 of the hot path), phase taken at the GRIDDED cell so that the weighted channel sum of a row is exactly
// the image pixel.  One CTA per (channel, row); lanes stride over baselines; float32 arithmetic.
#include <math_constants.h>

#include "rf_internal.h"

namespace rf {

namespace {

template <int NPOL>
__global__ void __launch_bounds__(128) k_cand_spectrum(const float* __restrict__ vis, const int32_t* __restrict__ delay_dm,
                                                       const int32_t* __restrict__ cell, const uint8_t* __restrict__ keep,
                                                       const float2* __restrict__ mean_i, int nint, int nbl, int nchan,
                                                       int npix, int dt, int j0, int maxdelay, int x, int y,
                                                       float* __restrict__ spec) {
    const int ch = blockIdx.x, r = blockIdx.y;
    const int jj = j0 + r;
    const bool in_range = jj >= 0 && (long long)(jj + 1) * dt + maxdelay <= nint;
    float acc = 0.f;
    int cnt = 0;
    const long long row_floats = (long long)nbl * nchan * NPOL * 2;
    const int t_first = jj * dt + delay_dm[ch];
    for (int bl = threadIdx.x; bl < nbl; bl += blockDim.x) {
        const size_t e = (size_t)bl * nchan + ch;
        if (!keep[e]) continue;
        cnt++;
        if (!in_range) continue;
        float re = 0.f, im = 0.f;
        for (int q = 0; q < dt; q++) {
            const float* s = vis + (long long)(t_first + q) * row_floats + e * (2 * NPOL);
#pragma unroll
            for (int pol = 0; pol < NPOL; pol++) { re += s[2 * pol]; im += s[2 * pol + 1]; }
        }
        if (mean_i != nullptr) { const float2 m = mean_i[e]; re -= (float)dt * m.x; im -= (float)dt * m.y; }
        const int k = (cell[2 * e] * x + cell[2 * e + 1] * y) & (npix - 1);      // npix is a power of two
        float sn, cs;
        sincospif(2.f * (float)k / (float)npix, &sn, &cs);
        acc += re * cs - im * sn;
    }
    __shared__ float s_acc[4];
    __shared__ int s_cnt[4];
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        acc += __shfl_xor_sync(0xffffffffu, acc, d);
        cnt += __shfl_xor_sync(0xffffffffu, cnt, d);
    }
    if ((threadIdx.x & 31) == 0) { s_acc[threadIdx.x >> 5] = acc; s_cnt[threadIdx.x >> 5] = cnt; }
    __syncthreads();
    if (threadIdx.x == 0) {
        const float a = (s_acc[0] + s_acc[1]) + (s_acc[2] + s_acc[3]);
        const int n = s_cnt[0] + s_cnt[1] + s_cnt[2] + s_cnt[3];
        spec[(size_t)r * nchan + ch] = n > 0 ? a / ((float)n * (float)dt * (float)NPOL) : 0.f;
    }
}

// Mock-transient injection ("randomly insert mock transient sources into data",
// PAPER.md:135; reading A18): vis[t0 + q + delay[ch]][bl][ch][pol] += A e^{-2 pi i (u l + v m) cell}, q < width,
// delay = the O1 expression at the injected DM (float64, explicit rounding, same operation order as
// k_delay_table); the phase is evaluated in float64 (up to ~100 turns), the sum is rounded once to float32.
// One thread per (baseline, channel); samples outside the segment are dropped.
__global__ void k_inject(float2* __restrict__ vis, const double* __restrict__ freqs_hz, const double* __restrict__ uvw,
                         int nint, int nbl, int nchan, int npol, double fmax_ghz, double inttime, double cell,
                         double amp, double l_pix, double m_pix, double dm, int width, int t0) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nbl * nchan) return;
    const int ch = i % nchan, bl = i / nchan;
    const double fh = freqs_hz[ch];
    const double f = __ddiv_rn(fh, 1e9);
    const double a = __ddiv_rn(1.0, __dmul_rn(f, f));
    const double b = __ddiv_rn(1.0, __dmul_rn(fmax_ghz, fmax_ghz));
    const double x = __ddiv_rn(__dmul_rn(__dmul_rn(4.148808e-3, dm), __dsub_rn(a, b)), inttime);
    const int delay = (int)floor(__dadd_rn(x, 0.5));
    const double ul = uvw[3 * bl + 0] * fh / 299792458.0, vl = uvw[3 * bl + 1] * fh / 299792458.0;
    double sn, cs;
    sincospi(-2.0 * (ul * l_pix + vl * m_pix) * cell, &sn, &cs);
    const double re = amp * cs, im = amp * sn;
    const size_t row = (size_t)nbl * nchan * npol;
    for (int q = 0; q < width; q++) {
        const long long t = (long long)t0 + q + delay;
        if (t < 0 || t >= nint) continue;
        float2* dst = vis + (size_t)t * row + (size_t)i * npol;
        for (int pol = 0; pol < npol; pol++) {
            float2 v = dst[pol];
            dst[pol] = make_float2((float)((double)v.x + re), (float)((double)v.y + im));
        }
    }
}

}  // namespace

int launch_inject(rf_plan* p, void* vis, double amp, double l_pix, double m_pix, double dm, int width, int t0,
                  cudaStream_t st) {
    double fmax = 0.0;
    for (double f : p->freqs) fmax = f > fmax ? f : fmax;
    const int n = p->nbl * p->nchan;
    k_inject<<<(n + 255) / 256, 256, 0, st>>>(reinterpret_cast<float2*>(vis), p->d.freqs, p->d.uvw, p->nint, p->nbl,
                                              p->nchan, p->npol, fmax / 1e9, p->inttime, p->cell, amp, l_pix, m_pix, dm,
                                              width, t0);
    RF_CUDA_CHECK(cudaGetLastError());
    return RF_OK;
}

int launch_cand_spectrum(rf_plan* p, const void* vis, int dm_idx, int dt_idx, int t_idx, int l_pix, int m_pix,
                         int half_window, float* spec_dev, cudaStream_t st) {
    int rc = RF_OK;
    if (p->meansub && (rc = launch_time_mean(p, vis, st)) != RF_OK) return rc;
    const int dt = p->dts[dt_idx];
    const int x = ((l_pix % p->npix) + p->npix) % p->npix, y = ((m_pix % p->npix) + p->npix) % p->npix;
    const dim3 grid(p->nchan, 2 * half_window + 1);
    const float* v = reinterpret_cast<const float*>(vis);
    const int32_t* drow = p->d.delay + (size_t)dm_idx * p->nchan;
    const float2* mi = p->meansub ? p->ws.mean_i : nullptr;
#define RF_SPEC(NPOL)                                                                                         \
    k_cand_spectrum<NPOL><<<grid, 128, 0, st>>>(v, drow, p->d.cell, p->d.keep, mi, p->nint, p->nbl, p->nchan, \
                                               p->npix, dt, t_idx - half_window, p->h_maxdelay[dm_idx], x, y, spec_dev)
    switch (p->npol) {
        case 1: RF_SPEC(1); break;
        case 2: RF_SPEC(2); break;
        default: RF_SPEC(4); break;
    }
#undef RF_SPEC
    RF_CUDA_CHECK(cudaGetLastError());
    return RF_OK;
}

}  // namespace rf
