// rf_kernels.cuh -- the two hot kernels of the search loop (sm_100a).
//
//   k_grid_colfft  : steps (b)+(c)+first half of (d): fused dedisperse + boxcar-resample read,
//                    Stokes-I sum, uv gridding into a shared-memory tile of uv columns (segmented
//                    warp sums, no atomics), inverse FFT along v of every column, transposed
//                    coalesced store of the half-plane H[y][c]; Parseval partial sums.
//   k_rowfft_stats : second half of (d) + (e): Hermitian row transform (two images per complex
//                    FFT), peak/argmax, shared-memory histogram -> median/MAD sigma, S/N,
//                    threshold and candidate compaction.
// Citations: PAPER.md:63, 88, 104, 118 (method); SURVEY.md 8a-2..8a-5 (layouts).
#pragma once
#include <cuda_runtime.h>
#include <math_constants.h>

#include "rf_fft.cuh"
#include "rf_internal.h"

namespace rf {

struct SearchParams {
    const float* vis;               // complex64 [nint][nbl][nchan][npol] as floats
    const float2* mean_i;           // [nbl*nchan] Stokes-I sum of the time means, or null (no subtraction)
    const float2* visI;             // [nbl*nchan][tpitch] time-fastest Stokes-I sums (mean already removed), or null
    int32_t tpitch;
    const int32_t* delay;           // [ndm][nchan]
    const GridEntry* entries;
    const int32_t* warp_chunk;
    const ImgDesc* images;          // first image of this batch
    const float2* twiddles;         // [16 + 256] per-stage FFT twiddles (rf_fft.cuh)
    float2* H;                      // [batch][N][cpad]
    float* sumsq;                   // [batch][ngroups]
    uint32_t* hist;                 // [batch][nbins]
    float* peak_val;                // [batch][rsplit]
    int32_t* peak_pos;
    uint32_t* ticket;               // [batch/2]
    int32_t* counters;
    rf_cand* cand_items;
    int32_t* cand_count;
    int32_t cand_capacity;
    float* image_out;               // debug: [N][N] image of batch slot 0 (or null)
    rf_cand* stats_out;             // debug: statistics of batch slot 0 (or null)
    int32_t nchan, ncol, cpad, ngroups, nbins, rsplit, n_img;
    long long row_floats;           // floats per integration = nbl*nchan*npol*2
    float norm;                     // 1 / (2 N_w npol)
    float threshold;
};

__device__ __forceinline__ float warp_sum(float x) {
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) x += __shfl_xor_sync(0xffffffffu, x, d);
    return x;
}


// Gather + segmented grid add for the chunk range [c_beg, c_end) of one warp.
// DT > 0: boxcar width known at compile time (fully unrolled); DT == 0: runtime width `dt`.
// U chunks are processed together so that U x DT independent loads are in flight per lane.
template <int NPOL, int DT, int U, int PITCH>
__device__ __forceinline__ void gather_grid(const SearchParams& p, float2* __restrict__ tile,
                                            const int* __restrict__ sdelay, const float* __restrict__ base,
                                            int c_beg, int c_end, int lane, int dt) {
    for (int ck = c_beg; ck < c_end; ck += U) {
        GridEntry e[U];
        const float* src[U];
        float re[U], im_[U];
#pragma unroll
        for (int u = 0; u < U; u++) {
            e[u] = (ck + u < c_end) ? p.entries[(size_t)(ck + u) * 32 + lane] : GridEntry{0u, 0u};
            re[u] = 0.f; im_[u] = 0.f;
        }
#pragma unroll
        for (int u = 0; u < U; u++)
            src[u] = base + (long long)sdelay[e[u].w1 & 0xfff] * p.row_floats + (size_t)(e[u].w0 & 0xffffffu) * (2 * NPOL);
        const int nq = DT > 0 ? DT : dt;
#pragma unroll
        for (int q = 0; q < nq; q++) {
#pragma unroll
            for (int u = 0; u < U; u++) {
                if (e[u].w0 >> 31) {
                    const float* s = src[u] + (long long)q * p.row_floats;
                    if (NPOL == 1) {
                        float2 a = __ldg(reinterpret_cast<const float2*>(s));
                        re[u] += a.x; im_[u] += a.y;
                    } else {
#pragma unroll
                        for (int h = 0; h < NPOL / 2; h++) {
                            float4 a = __ldg(reinterpret_cast<const float4*>(s) + h);
                            re[u] += a.x + a.z; im_[u] += a.y + a.w;
                        }
                    }
                }
            }
        }
        if (p.mean_i != nullptr) {     // mean-visibility subtraction: sum_q (x_q - m) = sum_q x_q - nq m
#pragma unroll
            for (int u = 0; u < U; u++) {
                if (e[u].w0 >> 31) {
                    const float2 m = __ldg(p.mean_i + (e[u].w0 & 0xffffffu));
                    re[u] = fmaf(-(float)nq, m.x, re[u]);
                    im_[u] = fmaf(-(float)nq, m.y, im_[u]);
                }
            }
        }
#pragma unroll
        for (int u = 0; u < U; u++) {
            if (e[u].w0 & (1u << 30)) im_[u] = -im_[u];
            // segmented inclusive scan: lanes of one cell are contiguous, `dist` = lanes to its head
            const int dist = (e[u].w0 >> 24) & 31;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                float r2 = __shfl_up_sync(0xffffffffu, re[u], d);
                float i2 = __shfl_up_sync(0xffffffffu, im_[u], d);
                if (dist >= d) { re[u] += r2; im_[u] += i2; }
            }
            if ((e[u].w0 >> 31) && (e[u].w0 & (1u << 29))) {
                const int row = (e[u].w1 >> 12) & 0xfff, col = (e[u].w1 >> 24) & 0xf;
                float2* dst = &tile[col * PITCH + fft_pad(row)];
                float2 cur = *dst;
                *dst = make_float2(cur.x + re[u], cur.y + im_[u]);
            }
            __syncwarp();
        }
    }
}

// The same gather from the time-fastest Stokes-I array of the boxcar-tree path (when the plan has one):
// the dt samples of an entry are contiguous (8*dt bytes) instead of dt scattered 16-byte pol pairs.
template <int PITCH>
__device__ __forceinline__ void gather_grid_visi(const SearchParams& p, float2* __restrict__ tile,
                                                 const int* __restrict__ sdelay, int t_first,
                                                 int c_beg, int c_end, int lane, int dt,
                                                 const float2* __restrict__ arr) {
    for (int ck = c_beg; ck < c_end; ck++) {
        const GridEntry e = p.entries[(size_t)ck * 32 + lane];
        const bool valid = (e.w0 >> 31) != 0;
        const float2* src = arr + (size_t)(e.w0 & 0xffffffu) * p.tpitch + (t_first + sdelay[e.w1 & 0xfff]);
        float re = 0.f, im = 0.f;
        if (valid) {
            int q = 0;
            for (; q + 8 <= dt; q += 8) {
                float2 a[8];
#pragma unroll
                for (int k = 0; k < 8; k++) a[k] = __ldg(src + q + k);
#pragma unroll
                for (int k = 0; k < 8; k++) { re += a[k].x; im += a[k].y; }
            }
            for (; q < dt; q++) { const float2 a = __ldg(src + q); re += a.x; im += a.y; }
        }
        if (e.w0 & (1u << 30)) im = -im;
        const int dist = (e.w0 >> 24) & 31;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            float r2 = __shfl_up_sync(0xffffffffu, re, d);
            float i2 = __shfl_up_sync(0xffffffffu, im, d);
            if (dist >= d) { re += r2; im += i2; }
        }
        if (valid && (e.w0 & (1u << 29))) {
            const int row = (e.w1 >> 12) & 0xfff, col = (e.w1 >> 24) & 0xf;
            float2* dst = &tile[col * PITCH + fft_pad(row)];
            float2 cur = *dst;
            *dst = make_float2(cur.x + re, cur.y + im);
        }
        __syncwarp();
    }
}

// ------------------------------------------------------------------------------------------
// Pass 1.  grid = (n_img, ngroups): group-major launch order, so the heavy central column
// groups start first (measured faster than image-major order); block = 256.  Dynamic smem:
//   tile  [NCOL][PITCH] float2, PITCH = fft_padded_size(N) + 1 (odd -> conflict-free transpose)
//   tw    [TW_TOTAL] float2 | sdelay [nchan] int | red [8] float
template <int N, int NPOL, int NCOL>
__global__ void __launch_bounds__(kThreads) k_grid_colfft(const SearchParams p) {
    using C = FftCfg<N>;
    constexpr int PITCH = fft_padded_size(N) + 1;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2* tile = reinterpret_cast<float2*>(smem_raw);
    float2* tw = tile + NCOL * PITCH;
    int* sdelay = reinterpret_cast<int*>(tw + C::TW_TOTAL);
    float* red = reinterpret_cast<float*>(sdelay + p.nchan);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int slot = blockIdx.x, g = blockIdx.y;
    const ImgDesc im = p.images[slot];

    for (int i = tid; i < NCOL * PITCH; i += kThreads) tile[i] = make_float2(0.f, 0.f);
    for (int i = tid; i < p.nchan; i += kThreads) sdelay[i] = p.delay[(size_t)im.dm_idx * p.nchan + i];
    load_twiddles<N>(tw, p.twiddles, tid, kThreads);
    __syncthreads();

    // ---- (b)+(c): gather at the delayed time index, boxcar + Stokes sum, segmented grid add
    {
        const int c_beg = p.warp_chunk[g * kWarpsPerCta + warp];
        const int c_end = p.warp_chunk[g * kWarpsPerCta + warp + 1];
        const float* base = p.vis + (long long)im.j * im.dt * p.row_floats;
        if (p.visI != nullptr) gather_grid_visi<PITCH>(p, tile, sdelay, im.j * im.dt, c_beg, c_end, lane, im.dt, p.visI);
        else switch (im.dt) {   // compile-time widths keep U x DT independent 16-byte loads in flight per lane
            case 1: gather_grid<NPOL, 1, 8, PITCH>(p, tile, sdelay, base, c_beg, c_end, lane, 1); break;
            case 2: gather_grid<NPOL, 2, 4, PITCH>(p, tile, sdelay, base, c_beg, c_end, lane, 2); break;
            case 4: gather_grid<NPOL, 4, 2, PITCH>(p, tile, sdelay, base, c_beg, c_end, lane, 4); break;
            case 8: gather_grid<NPOL, 8, 1, PITCH>(p, tile, sdelay, base, c_beg, c_end, lane, 8); break;
            default: gather_grid<NPOL, 0, 4, PITCH>(p, tile, sdelay, base, c_beg, c_end, lane, im.dt); break;
        }
    }
    __syncthreads();

    // ---- (d) first half: inverse FFT along v of each column, in place in the tile
    const float scale = p.norm / (float)im.dt;
    float ss = 0.f;
    {
        constexpr int G1 = kThreads / C::TPF;           // concurrent FFTs
        const int grp = tid / C::TPF, t = tid % C::TPF;
        for (int c = grp; c < NCOL; c += G1) {
            float2* col = tile + c * PITCH;
            float2 v[16];
            fft_reload<N>(v, col, t);
            const int gc = g * NCOL + c;
            const float wgt = (gc == 0 || gc == N / 2) ? 1.f : 2.f;
            float s = 0.f;
#pragma unroll
            for (int e = 0; e < 16; e++) s += v[e].x * v[e].x + v[e].y * v[e].y;
            ss += wgt * s;
            fft_inverse<N>(v, col, tw, t, 1 + grp);
            fft_group_sync<C::TPF>(1 + grp);            // all lanes done reading the exchange data
            fft_unload<N>(v, col, t, scale);
        }
    }
    ss = warp_sum(ss);
    if (lane == 0) red[warp] = ss;
    __syncthreads();
    if (tid == 0) {
        float tot = 0.f;
#pragma unroll
        for (int w = 0; w < kWarpsPerCta; w++) tot += red[w];
        p.sumsq[(size_t)slot * p.ngroups + g] = tot * scale * scale;
    }

    // ---- transposed store H[slot][y][g*NCOL + c]: NCOL*8 contiguous bytes per row
    {
        float2* Hs = p.H + (size_t)slot * N * p.cpad + g * NCOL;
        const int c = tid % NCOL, y0 = tid / NCOL;
        for (int y = y0; y < N; y += kThreads / NCOL)
            Hs[(size_t)y * p.cpad + c] = tile[c * PITCH + fft_pad(y)];
    }
}

// ------------------------------------------------------------------------------------------
// Interpolated cumulative count below x from a histogram with exclusive prefix sums.
struct HistView {
    const uint32_t* h;      // counts [nbins]
    const uint32_t* cum;    // exclusive prefix [nbins]
    int nbins;
    float lo, inv_w;
    __device__ __forceinline__ float below(float x) const {
        float pos = (x - lo) * inv_w;
        pos = fminf(fmaxf(pos, 0.f), (float)nbins);
        int b = min((int)pos, nbins - 1);
        return (float)cum[b] + (pos - (float)b) * (float)h[b];
    }
};

// Median and MAD of one image from its histogram; executed by warp 0 of the finalising CTA.
// Returns sigma (1.4826 * MAD) in lane 0; sets *overflow when a quantile sits in a clamp bin.
__device__ float robust_sigma_from_hist(const HistView& hv, float total, int lane, int* overflow) {
    const float target = 0.5f * total;
    // median: bin where the exclusive prefix crosses total/2 (binary search, all lanes redundantly)
    int lo_b = 0, hi_b = hv.nbins - 1;
    while (lo_b < hi_b) {
        int mid = (lo_b + hi_b + 1) >> 1;
        if ((float)hv.cum[mid] <= target) lo_b = mid; else hi_b = mid - 1;
    }
    const int bm = lo_b;
    const float hb = (float)hv.h[bm];
    const float w = 1.f / hv.inv_w;
    const float med = hv.lo + ((float)bm + (hb > 0.f ? (target - (float)hv.cum[bm]) / hb : 0.5f)) * w;
    // MAD: smallest m with below(med + m) - below(med - m) >= total/2; 33-section search per round
    float a = 0.f, b = (float)hv.nbins * w;
    for (int round = 0; round < 6; round++) {
        const float step = (b - a) * (1.f / 33.f);
        const float m = a + step * (float)(lane + 1);
        const float cnt = hv.below(med + m) - hv.below(med - m);
        const unsigned ge = __ballot_sync(0xffffffffu, cnt >= target);
        const int first = ge ? (__ffs(ge) - 1) : 32;      // first lane at or above the target
        const float na = a + step * (float)first;
        b = (first == 32) ? b : a + step * (float)(first + 1);
        a = na;
    }
    const float mad = 0.5f * (a + b);
    if (bm == 0 || bm == hv.nbins - 1) *overflow = 1;
    {
        float p1 = (med + mad - hv.lo) * hv.inv_w, p0 = (med - mad - hv.lo) * hv.inv_w;
        if (p1 >= (float)(hv.nbins - 1) || p0 < 1.f) *overflow = 1;
    }
    return 1.4826f * mad;
}


// ------------------------------------------------------------------------------------------
// Exact order statistics for images small enough to stay in shared memory (npix <= 128):
// MSB-first radix select on order-preserving keys, 4 passes of 8 bits, whole CTA.
__device__ __forceinline__ uint32_t float_key(float f) {
    uint32_t u = __float_as_uint(f);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float key_float(uint32_t k) {
    return __uint_as_float((k & 0x80000000u) ? (k & 0x7fffffffu) : ~k);
}
// k-th smallest (0-based) of data[0..M); h256 = 258 words of shared scratch.  All threads call.
__device__ float select_kth(const float* data, int M, int k, uint32_t* h256) {
    uint32_t prefix = 0u, mask = 0u;
    const int tid = threadIdx.x;
    for (int shift = 24; shift >= 0; shift -= 8) {
        __syncthreads();
        h256[tid] = 0u;                               // blockDim.x == 256
        __syncthreads();
        for (int i = tid; i < M; i += kThreads) {
            const uint32_t key = float_key(data[i]);
            if ((key & mask) == prefix) atomicAdd(&h256[(key >> shift) & 255u], 1u);
        }
        __syncthreads();
        if (tid == 0) {
            int cum = 0, d = 0;
            for (; d < 255; d++) {
                const int c = (int)h256[d];
                if (cum + c > k) break;
                cum += c;
            }
            h256[256] = (uint32_t)d;
            h256[257] = (uint32_t)(k - cum);
        }
        __syncthreads();
        prefix |= h256[256] << shift;
        k = (int)h256[257];
        mask |= 255u << shift;
    }
    __syncthreads();
    return key_float(prefix);
}
// 1.4826 * median(|x - median(x)|), numpy's even-count median (mean of the two middle values).
// Overwrites data with the absolute deviations.  All threads call; all get the result.
__device__ float exact_sigma(float* data, int M, uint32_t* h256) {
    const float med = 0.5f * (select_kth(data, M, M / 2 - 1, h256) + select_kth(data, M, M / 2, h256));
    for (int i = threadIdx.x; i < M; i += kThreads) data[i] = fabsf(data[i] - med);
    __syncthreads();
    const float mad = 0.5f * (select_kth(data, M, M / 2 - 1, h256) + select_kth(data, M, M / 2, h256));
    return 1.4826f * mad;
}

// ------------------------------------------------------------------------------------------
// Pass 2.  grid = (rsplit, npairs); block = 256.  Dynamic smem:
//   xbuf [G2][fft_padded_size(N)] float2 | tw | hist [2][nbins] u32 | cum [nbins] u32 | scratch
//   | (EXACT only) simg [2][N*N] float
// EXACT (npix <= 128, row split 1): the two images stay in shared memory and median / MAD are
// exact order statistics; otherwise they come from a 2048-bin histogram over +-3.5 sigma_rms.
template <int N, bool EXACT>
__global__ void __launch_bounds__(kThreads) k_rowfft_stats(const SearchParams p) {
    using C = FftCfg<N>;
    constexpr int G2 = kThreads / C::TPF;
    constexpr int XB = fft_padded_size(N);
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2* xbuf = reinterpret_cast<float2*>(smem_raw);
    float2* tw = xbuf + G2 * XB;
    uint32_t* hist = reinterpret_cast<uint32_t*>(tw + C::TW_TOTAL);   // [2][nbins]
    uint32_t* cum = hist + 2 * p.nbins;                               // [nbins]
    float* s_val = reinterpret_cast<float*>(cum + p.nbins);           // [2][8]
    int* s_pos = reinterpret_cast<int*>(s_val + 16);                  // [2][8]
    float* s_misc = reinterpret_cast<float*>(s_pos + 16);             // [8]
    int* s_flag = reinterpret_cast<int*>(s_misc + 8);                 // [4]
    float* simg = reinterpret_cast<float*>(s_flag + 4);               // [2][N*N] (EXACT)

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int pair = blockIdx.y, rs = blockIdx.x;
    const int slot_a = 2 * pair, slot_b = 2 * pair + 1;
    const bool has_b = slot_b < p.n_img;

    for (int i = tid; i < 2 * p.nbins; i += kThreads) hist[i] = 0u;
    load_twiddles<N>(tw, p.twiddles, tid, kThreads);
    // sigma_rms of both images from the Parseval partials (fixed summation order)
    if (tid < 2) {
        float tot = 0.f;
        const int slot = 2 * pair + tid;
        if (slot < p.n_img)
            for (int gidx = 0; gidx < p.ngroups; gidx++) tot += p.sumsq[(size_t)slot * p.ngroups + gidx];
        s_misc[tid] = sqrtf(tot);       // mean(img^2) = sum |G|^2 scale^2  (Parseval)
    }
    __syncthreads();
    const float sig_a = s_misc[0], sig_b = s_misc[1];
    const float lo_a = -kHistRange * sig_a, lo_b = -kHistRange * sig_b;
    const float iw_a = sig_a > 0.f ? (float)p.nbins / (2.f * kHistRange * sig_a) : 0.f;
    const float iw_b = sig_b > 0.f ? (float)p.nbins / (2.f * kHistRange * sig_b) : 0.f;
    const unsigned nbm1 = (unsigned)p.nbins - 1u;

    const float2* Ha = p.H + (size_t)slot_a * N * p.cpad;
    const float2* Hb = p.H + (size_t)(has_b ? slot_b : slot_a) * N * p.cpad;
    const int grp = tid / C::TPF, t = tid % C::TPF;
    float2* xb = xbuf + grp * XB;
    const int rows = N / p.rsplit, y_beg = rs * rows;

    float best_a = -CUDART_INF_F, best_b = -CUDART_INF_F;
    int pos_a = 0, pos_b = 0;

    for (int y = y_beg + grp; y < y_beg + rows; y += G2) {
        const float2* ra = Ha + (size_t)y * p.cpad;
        const float2* rb = Hb + (size_t)y * p.cpad;
        float2 v[16];
        // Z[c] = Ha[c] + i Hb[c] (c >= 0);  Z[N - c] = conj(Ha[c]) + i conj(Hb[c])
#pragma unroll
        for (int e = 0; e < 16; e++) {
            const int c = t + C::TPF * e;
            const int cc = (e < 8) ? c : N - c;          // e == 8, t == 0 -> cc = N/2
            float2 a = make_float2(0.f, 0.f), b = make_float2(0.f, 0.f);
            if (cc < p.ncol) {
                a = ra[cc];
                if (has_b) b = rb[cc];
            }
            if (cc == 0 || cc == N / 2) v[e] = make_float2(a.x, b.x);
            else if (e < 8) v[e] = make_float2(a.x - b.y, a.y + b.x);
            else v[e] = make_float2(a.x + b.y, b.x - a.y);
        }
        fft_inverse<N>(v, xb, tw, t, 1 + grp);
        // ---- (e) statistics straight from registers
        float ma = v[0].x, mb = v[0].y;
#pragma unroll
        for (int e = 1; e < 16; e++) { ma = fmaxf(ma, v[e].x); mb = fmaxf(mb, v[e].y); }
        if (ma > best_a) {
            best_a = ma;
#pragma unroll
            for (int e = 15; e >= 0; e--) if (v[e].x == ma) pos_a = y * N + t + C::TPF * e;
        }
        if (mb > best_b) {
            best_b = mb;
#pragma unroll
            for (int e = 15; e >= 0; e--) if (v[e].y == mb) pos_b = y * N + t + C::TPF * e;
        }
        if (EXACT) {
#pragma unroll
            for (int e = 0; e < 16; e++) {
                simg[y * N + t + C::TPF * e] = v[e].x;
                simg[N * N + y * N + t + C::TPF * e] = v[e].y;
            }
        } else {
            if (iw_a > 0.f) {
#pragma unroll
                for (int e = 0; e < 16; e++) {
                    const unsigned bin = __float2uint_rd((v[e].x - lo_a) * iw_a);   // saturates below 0
                    atomicAdd(&hist[min(bin, nbm1)], 1u);
                }
            }
            if (has_b && iw_b > 0.f) {
#pragma unroll
                for (int e = 0; e < 16; e++) {
                    const unsigned bin = __float2uint_rd((v[e].y - lo_b) * iw_b);
                    atomicAdd(&hist[p.nbins + min(bin, nbm1)], 1u);
                }
            }
        }
        if (p.image_out != nullptr && pair == 0) {
#pragma unroll
            for (int e = 0; e < 16; e++) p.image_out[(size_t)y * N + t + C::TPF * e] = v[e].x;
        }
    }

    // ---- CTA-wide peak (max value, smallest position on ties)
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        float ov = __shfl_xor_sync(0xffffffffu, best_a, d);
        int op = __shfl_xor_sync(0xffffffffu, pos_a, d);
        if (ov > best_a || (ov == best_a && op < pos_a)) { best_a = ov; pos_a = op; }
        ov = __shfl_xor_sync(0xffffffffu, best_b, d);
        op = __shfl_xor_sync(0xffffffffu, pos_b, d);
        if (ov > best_b || (ov == best_b && op < pos_b)) { best_b = ov; pos_b = op; }
    }
    if (lane == 0) { s_val[warp] = best_a; s_pos[warp] = pos_a; s_val[8 + warp] = best_b; s_pos[8 + warp] = pos_b; }
    __syncthreads();
    if (tid < 2) {
        float bv = s_val[8 * tid];
        int bp = s_pos[8 * tid];
        for (int w = 1; w < kWarpsPerCta; w++) {
            float ov = s_val[8 * tid + w];
            int op = s_pos[8 * tid + w];
            if (ov > bv || (ov == bv && op < bp)) { bv = ov; bp = op; }
        }
        s_val[8 * tid] = bv; s_pos[8 * tid] = bp;
    }
    __syncthreads();

    // ---- merge across the row split; the last CTA of the pair finalises
    if (!EXACT && p.rsplit > 1) {
        for (int i = tid; i < 2 * p.nbins; i += kThreads) {
            const uint32_t c = hist[i];
            if (c) atomicAdd(&p.hist[(size_t)slot_a * p.nbins + i], c);   // slots a, b are adjacent
        }
        if (tid < 2 && (tid == 0 || has_b)) {
            p.peak_val[(size_t)(slot_a + tid) * p.rsplit + rs] = s_val[8 * tid];
            p.peak_pos[(size_t)(slot_a + tid) * p.rsplit + rs] = s_pos[8 * tid];
        }
        __threadfence();
        __syncthreads();
        if (tid == 0) s_flag[0] = (atomicAdd(&p.ticket[pair], 1u) == (uint32_t)(p.rsplit - 1));
        __syncthreads();
        if (!s_flag[0]) return;
        __threadfence();
        for (int i = tid; i < 2 * p.nbins; i += kThreads) {
            uint32_t* gp = &p.hist[(size_t)slot_a * p.nbins + i];
            hist[i] = __ldcg(gp);
            *gp = 0u;                                   // self-cleaning for the next batch
        }
        if (tid < 2 && (tid == 0 || has_b)) {
            float bv = -CUDART_INF_F;
            int bp = 0;
            for (int r = 0; r < p.rsplit; r++) {
                float ov = __ldcg(&p.peak_val[(size_t)(slot_a + tid) * p.rsplit + r]);
                int op = __ldcg(&p.peak_pos[(size_t)(slot_a + tid) * p.rsplit + r]);
                if (ov > bv || (ov == bv && op < bp)) { bv = ov; bp = op; }
            }
            s_val[8 * tid] = bv; s_pos[8 * tid] = bp;
        }
        if (tid == 0) p.ticket[pair] = 0u;
        __syncthreads();
    }

    // ---- median / MAD / S/N / threshold, one image at a time
    for (int which = 0; which < (has_b ? 2 : 1); which++) {
        const uint32_t* h = hist + which * p.nbins;
        float sigma_exact = 0.f;
        if (EXACT) {
            sigma_exact = exact_sigma(simg + which * N * N, N * N, cum);
        } else {
            // exclusive prefix sum of nbins counters: per-thread chunk + warp scan + warp totals
            const int per = p.nbins / kThreads;             // nbins is a multiple of 256
            uint32_t local = 0;
            for (int i = 0; i < per; i++) local += h[tid * per + i];
            uint32_t inc = local;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                uint32_t o = __shfl_up_sync(0xffffffffu, inc, d);
                if (lane >= d) inc += o;
            }
            __shared__ uint32_t wtot[kWarpsPerCta];
            if (lane == 31) wtot[warp] = inc;
            __syncthreads();
            uint32_t base = inc - local;
            for (int w = 0; w < warp; w++) base += wtot[w];
            for (int i = 0; i < per; i++) { cum[tid * per + i] = base; base += h[tid * per + i]; }
            __syncthreads();
        }
        if (warp == 0) {
            const float sig_rms = which ? sig_b : sig_a;
            int overflow = 0;
            float sigma = 0.f;
            if (EXACT) {
                sigma = sigma_exact;
            } else if (sig_rms > 0.f) {
                HistView hv{h, cum, p.nbins, -kHistRange * sig_rms, (float)p.nbins / (2.f * kHistRange * sig_rms)};
                sigma = robust_sigma_from_hist(hv, (float)N * (float)N, lane, &overflow);
            }
            if (lane == 0) {
                const float peak = s_val[8 * which];
                const int pos = s_pos[8 * which];
                const float snr = sigma > 0.f ? peak / sigma : 0.f;
                const ImgDesc im = p.images[slot_a + which];
                int x = pos % N, yy = pos / N;
                rf_cand c;
                c.dm_idx = im.dm_idx; c.dt_idx = im.dt_idx; c.t_idx = im.j;
                c.l_pix = x < N / 2 ? x : x - N;
                c.m_pix = yy < N / 2 ? yy : yy - N;
                c.peak = peak; c.sigma = sigma; c.snr = snr;
                if (overflow) atomicAdd(&p.counters[0], 1);
                if (p.stats_out != nullptr && slot_a + which == 0) *p.stats_out = c;
                if (p.cand_count != nullptr) atomicAdd(&p.counters[1], 1);   // images finalised (rf_counters.images)
                // an all-zero image (sigma = 0) has snr := 0 and is never a candidate (reading A24)
                if (p.cand_count != nullptr && sigma > 0.f && snr >= p.threshold) {
                    int idx = atomicAdd(p.cand_count, 1);
                    if (idx < p.cand_capacity) p.cand_items[idx] = c;
                }
            }
        }
        __syncthreads();
    }
}

}  // namespace rf
