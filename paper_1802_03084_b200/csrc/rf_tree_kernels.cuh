// rf_tree_kernels.cuh -- the "boxcar tree" variant of the hot kernels (sm_100a).
//
// Gridding and the FFT are linear and the uv cell of a (baseline, channel) does not depend on
// time, so the image of (dm, dt, j) is the mean of the dt = 1 images j*dt .. j*dt+dt-1 of the same
// DM (SURVEY.md section 7 "boxcar linearity"; oracle pin P11).  For power-of-two widths the loops
// over sampling time and integration (Fig. 2) are therefore walked in BLOCKS of TB
// consecutive native integrations of one DM:
//
//   k_stokes_transpose   : vis [t][bl][ch][pol] -> Stokes-I sum visI [bl*nchan+ch][t] (time fastest),
//                          so a block reads TB*8 contiguous bytes per (baseline, channel).
//   k_tree_gather        : gathers the TB dedispersed samples of every entry and sums them per uv cell
//                          (compact grid of the occupied half-plane cells), Parseval sums of every tree node.
//   k_tree_colfft        : scatters the cells of its uv columns into shared-memory tiles, column FFTs,
//                          store of the half plane as H[y][pair][c][q & 1] (q = integration in the block).
//   k_tree_rowfft_stats  : per row, TB/2 Hermitian pair transforms; the wider images are running
//                          sums of the rows in registers; all 2*TB-1 images get peak, histogram,
//                          median/MAD, S/N and the threshold test.  The image is never stored.
#pragma once
#include <cuda_runtime.h>
#include <math_constants.h>

#include "rf_kernels.cuh"

namespace rf {

struct TreeParams {
    const float2* visI;             // [nbl*nchan][tpitch]
    const int32_t* delay;           // [ndm][nchan]
    const uint2* entries;           // gather entries, [n_iters][LG]
    const int32_t* stream_iter;     // [n_streams][2] first and past-the-last iteration of each warp stream (sorted by length)
    const int32_t* stream_cell;     // [n_streams] first cell of each warp stream
    const uint32_t* cells;          // [n_cells]
    const int32_t* group_cell;      // [ngroups + 1]
    const BlockDesc* blocks;        // first block of this batch
    const float2* twiddles;
    const float2* twp;              // [16][15] stage-2 twiddle powers (rf_fft.cuh), sizes >= 256
    float2* cellsum;                // [n_blk][n_cells][TB] compact grid (unscaled sums)
    float2* Ht;                     // [n_blk][N][TB/2][cpad][2]
    float* sumsq;                   // [n_blk][2*TB-1][n_parts]
    int32_t* counters;
    rf_cand* cand_items;
    int32_t* cand_count;
    int32_t cand_capacity;
    float* image_out;               // debug: image `dbg_img` of block 0
    rf_cand* stats_out;
    int32_t dbg_img;                // -1 = off
    int32_t dbg_slot;               // block of the launch the debug outputs refer to
    int32_t tpitch, nchan, ncol, cpad, ngroups, nbins, n_blk, n_cells, n_streams, n_parts;
    int32_t ncmax;                  // most cells in one column group (k_tree_coldft's value buffers)
    int32_t dft_max_blk;            // ints in the longest list block
    const int32_t* dft_blk;         // k_tree_coldft: list blocks of all column groups (rf_tables.cu)
    const int32_t* dft_off;         // [ngroups + 1] first int of each block (multiples of 4)
    int32_t part_major;             // gather grid (host side): 1 = x runs over block pairs, y over cell ranges, 0 = x over cell ranges
    int32_t dec;                    // 1, or the width dt whose phase-decimated sum array visI points at (B7)
    uint32_t phase_stride;          // dec > 1: elements per phase = (nbl*nchan + 1) * row pitch
    int32_t zero_row;               // >= 0: periodicity mode, every block uses this (all-zero) delay row
    long long slab_stride;          // periodicity mode: visI is [slab][nbl*nchan][tpitch], block.pad = slab
    int32_t dt_idx[4];              // tree level -> index in dt_list, or -1
    float norm;                     // 1 / (2 N_w npol)
    float threshold;
};

// image index of tree node (level l, i) inside a block: levels are stored one after the other
__host__ __device__ constexpr int tree_off(int tb, int l) {
    int off = 0;
    for (int m = 0; m < l; m++) off += tb >> m;
    return off;
}

// ------------------------------------------------------------------------------------------
// Stokes-I sum and transpose to time-fastest order.  grid (ceil(E/32), ceil(tpitch/32)), block (32, 8).
// Rows t >= nint of the output (the read-ahead pad of the last block) are zero.  mean_i (or null):
// Stokes-I sum of the time means, subtracted on the fly (mean-visibility subtraction).
template <int NPOL>
__global__ void k_stokes_transpose(const float* __restrict__ vis, float2* __restrict__ visI,
                                   const float2* __restrict__ mean_i, int nint, int nelem, int tpitch, int t_first) {
    __shared__ float2 tile[32][33];
    const int e0 = blockIdx.x * 32, t0 = t_first + blockIdx.y * 32;    // t_first: row range of a chunked upload
    for (int r = threadIdx.y; r < 32; r += 8) {
        const int t = t0 + r, e = e0 + threadIdx.x;
        float2 s = make_float2(0.f, 0.f);
        if (t < nint && e < nelem) {
            const float* src = vis + ((size_t)t * nelem + e) * (2 * NPOL);
            if (NPOL == 1) {
                s = *reinterpret_cast<const float2*>(src);
            } else {
#pragma unroll
                for (int h = 0; h < NPOL / 2; h++) {
                    float4 a = __ldg(reinterpret_cast<const float4*>(src) + h);
                    s.x += a.x + a.z; s.y += a.y + a.w;
                }
            }
            if (mean_i != nullptr) { const float2 m = __ldg(mean_i + e); s.x -= m.x; s.y -= m.y; }
        }
        tile[r][threadIdx.x] = s;
    }
    __syncthreads();
    for (int r = threadIdx.y; r < 32; r += 8) {
        const int e = e0 + r, t = t0 + threadIdx.x;
        if (e < nelem && t < tpitch) visI[(size_t)e * tpitch + t] = tile[threadIdx.x][r];
    }
}

// Phase-decimated boxcar sums of the time-fastest Stokes-I array for a width dt that is not on the tree (B7):
//   out[(phase * (nelem + 1) + e) * pitch + jp] = sum_{q < dt} visI[e][phase + dt * jp + q]     (0 past the array),
// i.e. the dt-sample boxcar starting at every integration t = phase + dt * jp, stored so that the boxcars one width
// apart are adjacent.  The dedispersed output integration j of a channel with delay d is the boxcar at t = d + dt j
// = element (phase d % dt, jp = j + d / dt): consecutive j are contiguous, so the tree gather reads them like native
// integrations.  grid (nelem, ceil(pitch / JC)), block 256; one CTA = one series x JC output integrations of every
// phase = a span of JC * dt native integrations staged in shared memory (coalesced read), boxcars formed from
// shared memory, written phase by phase in runs of JC contiguous values.  Dynamic smem: in [JC*dt + dt] | sums
// [JC*dt, padded by 1/32] float2.  The all-zero series of every phase is never written.
__global__ void __launch_bounds__(256) k_phase_sum(const float2* __restrict__ visI, float2* __restrict__ out,
                                                   int dt, int tpitch, int pitch, int nelem, int JC) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int span = JC * dt;
    float2* in = reinterpret_cast<float2*>(smem_raw);
    float2* sums = in + span + dt;
    const int e = blockIdx.x, j0 = blockIdx.y * JC, t0 = j0 * dt, tid = threadIdx.x;
    const float2* src = visI + (size_t)e * tpitch;
    for (int i = tid; i < span + dt; i += 256) in[i] = (t0 + i < tpitch) ? __ldg(src + t0 + i) : make_float2(0.f, 0.f);
    __syncthreads();
    for (int i = tid; i < span; i += 256) {
        float re = 0.f, im = 0.f;
        for (int q = 0; q < dt; q++) { re += in[i + q].x; im += in[i + q].y; }
        sums[i + (i >> 5)] = make_float2(re, im);
    }
    __syncthreads();
    for (int idx = tid; idx < span; idx += 256) {
        const int phase = idx / JC, i = idx % JC, jp = j0 + i;
        const int k = phase + dt * i;
        if (jp < pitch) out[((size_t)phase * (nelem + 1) + e) * pitch + jp] = sums[k + (k >> 5)];
    }
}

// ------------------------------------------------------------------------------------------
// Tree pass 0: gather + grid.  grid = (n_blk / GB, n_parts) [cell-range major] with GB = kGatherBlocks = 2; block = 256
// = 8 warp streams.  Dynamic smem:  sdelay [nchan] int | red [8][GB][2*TB-1] float.
// One CTA serves GB consecutive time blocks of one DM: slots GB y ... GB y + GB - 1 of the launch (build_image_list),
// i.e. GB TB consecutive integrations.
// "Time in lanes": lane = (entry j = lane / (GB TB), block h = (lane / TB) % GB, integration q = lane % TB).
// One iteration reads LG = 32 / (GB TB) entries; the GB TB dedispersed samples of an entry are ONE coalesced 8 GB TB-byte
// read of visI[bl*nchan + ch][t0 + delay[ch] + 0 .. GB TB - 1] (TB = 8, GB = 2: 128 bytes; the delay is arbitrary, so a run
// straddles one more 128-byte line than it fills).
// The lane accumulates over the iterations of a cell in a
// register; the END iteration sums the LG lane groups with xor shuffles and group 0 writes the cell
// sum (TB contiguous complex values per block) to the compact grid.  Parseval sums of every boxcar-tree node,
// sum_cells w |sum_{q in node} G_q|^2, are taken at the same place (another log2(TB) xor steps over
// q), so sigma_rms of every image of the block is known before any pixel exists.
// No tile, no barriers inside the loop, few registers: latency is hidden by occupancy.
template <int TB, bool PART_MAJOR>
__global__ void __launch_bounds__(kThreads, 4) k_tree_gather(const TreeParams p) {
    constexpr int NIMG = 2 * TB - 1;
    constexpr int GB = kGatherBlocks, LG = 32 / (GB * TB), U = kTreeUnroll;
    constexpr int LEVELS = (TB == 8) ? 4 : (TB == 4 ? 3 : 2);      // log2(TB) + 1
    extern __shared__ __align__(16) unsigned char smem_raw[];
    int* sdelay = reinterpret_cast<int*>(smem_raw);
    float* red = reinterpret_cast<float*>(sdelay + p.nchan);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    // the blocks slot ... slot + GB - 1.  part_major: consecutive CTAs serve the SAME cell range (= the same (baseline, channel)
    // series) for consecutive block pairs, whose windows overlap almost entirely (neighbouring DM trials, consecutive
    // times), so a series is fetched from HBM once per launch instead of once per pair
    const int part = PART_MAJOR ? blockIdx.y : blockIdx.x, slot = GB * (PART_MAJOR ? blockIdx.x : blockIdx.y);
    const BlockDesc blk = p.blocks[slot];
    const int j = lane / (GB * TB), h = (lane / TB) % GB, q = lane % TB;
    const int s = part * kWarpsPerCta + warp;
    const bool has = s < p.n_streams;
    const int it_beg = has ? p.stream_iter[2 * s] : 0;
    const int it_end = has ? p.stream_iter[2 * s + 1] : 0;
    int cell = has ? p.stream_cell[s] : 0;
    const int32_t* drow = p.delay + (size_t)(p.zero_row >= 0 ? p.zero_row : blk.dm_idx) * p.nchan;
    uint2 en[U];                           // entries of the next batch of iterations (prefetched)
#pragma unroll
    for (int u = 0; u < U; u++) en[u] = make_uint2(0u, 0u);
    if (it_beg < it_end) {
#pragma unroll
        for (int u = 0; u < U; u++) en[u] = p.entries[(size_t)(it_beg + u) * LG + j];
    }
    // dec > 1: integration t = delay + dt j of a series lives at (phase t % dt, output integration t / dt), so the
    // "delay" added to an entry's row offset is (delay % dt) * phase_stride + delay / dt and the block's TB (2 TB)
    // consecutive OUTPUT integrations are contiguous
    for (int i = tid; i < p.nchan; i += kThreads) {
        const int d = drow[i];
        sdelay[i] = p.dec > 1 ? (int)((uint32_t)(d % p.dec) * p.phase_stride + (uint32_t)(d / p.dec)) : d;
    }
    __syncthreads();

    float ps[LEVELS];
#pragma unroll
    for (int l = 0; l < LEVELS; l++) ps[l] = 0.f;
    // the sample of entry (x, y) is vbase[x + delay[channel(y)]]: one 32-bit add, one 64-bit scaled add
    const float2* vbase = p.visI + (size_t)blk.pad * p.slab_stride + blk.tb * TB + h * TB + q;
    asm volatile("" : "+l"(vbase));     // one register pointer: a sample's address is then a single 32 x 8 + 64-bit multiply-add
    float2* cs = p.cellsum + (size_t)(slot + h) * p.n_cells * TB + q;
    float2 acc = make_float2(0.f, 0.f);
    for (int it = it_beg; it < it_end; it += U) {
        uint32_t e[U];
        float2 x[U];
#pragma unroll
        for (int u = 0; u < U; u++) {
            e[u] = en[u].y;
            x[u] = __ldg(vbase + (en[u].x + (uint32_t)sdelay[en[u].y & 0xfffu]));
        }
        if (it + U < it_end) {
#pragma unroll
            for (int u = 0; u < U; u++) en[u] = p.entries[(size_t)(it + U + u) * LG + j];
        }
#pragma unroll
        for (int u = 0; u < U; u++) {
            acc.x += x[u].x;                                              // padding entries read zeros
            acc.y += __uint_as_float(__float_as_uint(x[u].y) ^ (e[u] & 0x80000000u));     // conjugate: bit 31
            if (e[u] & (1u << 29)) {                                      // warp-uniform: cell complete
#pragma unroll
                for (int d = GB * TB; d < 32; d <<= 1) {
                    acc.x += __shfl_xor_sync(0xffffffffu, acc.x, d);
                    acc.y += __shfl_xor_sync(0xffffffffu, acc.y, d);
                }
                if (j == 0) cs[(size_t)cell * TB] = acc;
                cell++;
                const float wgt = (e[u] & (1u << 28)) ? 1.f : 2.f;
                ps[0] = fmaf(wgt, acc.x * acc.x + acc.y * acc.y, ps[0]);
#pragma unroll
                for (int l = 1; l < LEVELS; l++) {
                    acc.x += __shfl_xor_sync(0xffffffffu, acc.x, 1 << (l - 1));
                    acc.y += __shfl_xor_sync(0xffffffffu, acc.y, 1 << (l - 1));
                    ps[l] = fmaf(wgt, acc.x * acc.x + acc.y * acc.y, ps[l]);
                }
                acc = make_float2(0.f, 0.f);
            }
        }
    }
    // node (level l, i) of block h is held by the lanes of group 0 with q >> l == i (all of them hold the same sum)
    if (j == 0) {
#pragma unroll
        for (int l = 0; l < LEVELS; l++)
            if ((q & ((1 << l) - 1)) == 0) red[(warp * GB + h) * NIMG + tree_off(TB, l) + (q >> l)] = ps[l];
    }
    __syncthreads();
    if (tid < GB * NIMG) {
        const int hh = tid / NIMG, node = tid % NIMG;
        float tot = 0.f;
#pragma unroll
        for (int w = 0; w < kWarpsPerCta; w++) tot += red[(w * GB + hh) * NIMG + node];
        p.sumsq[((size_t)(slot + hh) * NIMG + node) * p.n_parts + part] = tot * p.norm * p.norm;
    }
}

// ------------------------------------------------------------------------------------------
// Tree pass 1: column FFTs.  grid = (ngroups, n_blk, TB/QH) -- the column groups of one block run together,
// so their 32-byte pieces of one H line meet in L2 before the line is written back; block = NTH.
// Dynamic smem:  tile [QH*NCOL][PITCH] float2 (column f = q*NCOL + c) | tw | occ [QH*NCOL][N/16] u32
// The CTA scatters the cells of its NCOL uv columns, for QH of the block's TB integrations
// (blockIdx.z selects which: QH < TB keeps two columns per CTA, i.e. whole 32-byte sectors in the
// store, with tiles small enough for four CTAs per SM), from the compact grid into its tiles,
// transforms the QH*NCOL columns in place (inverse, along v) and stores the half plane.
// Entry (16 bytes = the two integrations of one (row, column)) of a double row in the row-pair hand-off: the two
// rows of a column share one 32-byte sector, and columns whose bit 2 is set hold them in swapped order, so that the
// row pass's 16-byte shared-memory reads of 8 consecutive columns of ONE row fall into 8 different bank groups
// (plain order: lane stride 32 bytes = 2-way bank conflicts on every staging read, +10 % on the 4096^2 row pass).
__host__ __device__ __forceinline__ int rp_entry(int c, int row_parity) { return 2 * c + (row_parity ^ ((c >> 2) & 1)); }

// RP ("row-pair" hand-off, N >= 2048 with TB = 2): H[slot][y / 2][c][y & 1][q] -- the two integrations of TWO
// consecutive rows of one column are 32 contiguous bytes, so a CTA that holds ONE column (two 4096-point tiles, 74 KB,
// three CTAs per SM instead of one) still writes whole 32-byte sectors, and a double row is contiguous for the row pass.
template <int N, int TB, int NCOL, int QH, int NTH, bool RP = false>
__global__ void __launch_bounds__(NTH) k_tree_colfft(const TreeParams p) {
    using C = FftCfg<N>;
    constexpr int PITCH = fft_padded_size(N) + 1;
    constexpr int NF = QH * NCOL;
    constexpr int KPRE = 3;                // compact-grid values per thread loaded before shared memory is touched
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2* tile = reinterpret_cast<float2*>(smem_raw);
    float2* tw = tile + NF * PITCH;
    uint32_t* occ = reinterpret_cast<uint32_t*>(tw + C::TW_TOTAL);   // [NF][TPF]: bit e = row t + TPF*e of the tile is set

    const int tid = threadIdx.x;
    const int g = blockIdx.x, slot = blockIdx.y, q0 = blockIdx.z * QH;
    const int c_beg = p.group_cell[g], c_end = p.group_cell[g + 1];
    const int nval = (c_end - c_beg) * QH;
    const float2* cs = p.cellsum + ((size_t)slot * p.n_cells + c_beg) * TB + q0;
    const uint32_t* cm = p.cells + c_beg;

    // ---- prologue: every global load of the set-up is issued before shared memory is touched
    const float2 tw0 = p.twiddles[tid < C::TW_TOTAL ? tid : 0];
    const float2 tw1 = p.twiddles[tid + NTH < C::TW_TOTAL ? tid + NTH : 0];
    float2 pv[KPRE];
    uint32_t pm[KPRE];
#pragma unroll
    for (int k = 0; k < KPRE; k++) {
        const int i = tid + k * NTH;
        pv[k] = make_float2(0.f, 0.f);
        pm[k] = 0u;
        if (i < nval) { pv[k] = cs[(i / QH) * TB + i % QH]; pm[k] = cm[i / QH]; }
    }
    // The tiles are NOT cleared: a column holds a few dozen occupied cells, so each (tile, thread) keeps a 16-bit
    // occupancy mask of its 16 rows and the transform loads only the rows that were written (the rest are zeros
    // in registers).  Saves the 70 KB clear and most of the first shared-memory read of every CTA.
    for (int i = tid; i < NF * C::TPF; i += NTH) occ[i] = 0u;
    if (tid < C::TW_TOTAL) tw[tid] = tw0;
    if (tid + NTH < C::TW_TOTAL) tw[tid + NTH] = tw1;
    __syncthreads();
    // ---- scatter the cells of these columns: value i = (cell i / QH, integration q0 + i % QH)
    auto put = [&](int i, uint32_t m, float2 val) {
        const int f = (i % QH) * NCOL + ((m >> 12) & 0xf), row = m & 0xfff;
        tile[f * PITCH + fft_pad(row)] = val;
        atomicOr(&occ[f * C::TPF + row % C::TPF], 1u << (row / C::TPF));
    };
#pragma unroll
    for (int k = 0; k < KPRE; k++) {
        const int i = tid + k * NTH;
        if (i < nval) put(i, pm[k], pv[k]);
    }
    for (int i = tid + KPRE * NTH; i < nval; i += NTH) put(i, cm[i / QH], cs[(i / QH) * TB + i % QH]);
    __syncthreads();

    // ---- column FFTs in place (inverse, along v)
    {
        constexpr int G1 = NTH / C::TPF;
        const int grp = tid / C::TPF, t = tid % C::TPF;
        for (int f = grp; f < NF; f += G1) {
            float2* col = tile + f * PITCH;
            float2 v[16];
            const uint32_t m = occ[f * C::TPF + t];
#pragma unroll
            for (int e = 0; e < 16; e++) {
                v[e] = make_float2(0.f, 0.f);
                if ((m >> e) & 1u) v[e] = col[fft_pad(t + C::TPF * e)];
            }
            fft_inverse<N>(v, col, tw, t, 1 + grp);
            fft_group_sync<C::TPF>(1 + grp);
            fft_unload<N>(v, col, t, p.norm);
        }
    }
    __syncthreads();

    // ---- store H[slot][y][pair][g*NCOL + c][q & 1] (pair = q / 2): the two integrations that share
    //      one Hermitian pair transform are adjacent (one 16-byte store), and one (row, pair) is
    //      contiguous for pass 2
    {
        constexpr int SEG = NCOL * QH / 2;
        float4* Hs = reinterpret_cast<float4*>(p.Ht + (size_t)slot * N * p.cpad * TB);
        // Row of each thread within the NTH/SEG rows of an iteration: a bit permutation of tid / SEG chosen so that
        // the 16 lanes of a half-warp (16/SEG rows x SEG tiles, tile pitch = 1 mod 16 words) read 16 different
        // 8-byte bank pairs (identity order: 2-way conflicts, rows y and y + 1 collide on neighbouring tiles).
        int y0 = tid / SEG;
        if (SEG == 8) y0 = (y0 & ~3) | ((y0 & 1) << 1) | ((y0 >> 1) & 1);
        else if (SEG == 4) y0 = (y0 & ~15) | ((y0 & 1) << 1) | ((y0 & 2) << 2) | ((y0 >> 2) & 1) | ((y0 & 8) >> 1);
        else if (SEG == 2) y0 = (y0 & ~15) | ((y0 & 7) << 1) | ((y0 >> 3) & 1);
        const int i = tid % SEG, pr = i / NCOL, c = i % NCOL;
        const float2* ta = tile + (2 * pr * NCOL + c) * PITCH;
        const float2* tb = ta + NCOL * PITCH;
        const bool col0 = g * NCOL + c == 0;
        for (int y = y0; y < N; y += NTH / SEG) {
            float2 a = ta[fft_pad(y)], b = tb[fft_pad(y)];
            if (col0) { a.y = 0.f; b.y = 0.f; }       // column 0 is Hermitian along v: its transform is real (B2)
            if (RP) Hs[(((size_t)(y >> 1)) * (TB / 2) + q0 / 2 + pr) * p.cpad * 2 + rp_entry(g * NCOL + c, y & 1)] = make_float4(a.x, a.y, b.x, b.y);
            else Hs[((size_t)y * (TB / 2) + q0 / 2 + pr) * p.cpad + g * NCOL + c] = make_float4(a.x, a.y, b.x, b.y);
        }
    }
}

// ------------------------------------------------------------------------------------------
// Tree pass 2.  grid = (n_blk); block = 256; one CTA = all rows of one block.  Dynamic smem:
//   xbuf [G2][XB] float2 (reused after the row loop for the unpacked histogram + prefix sums)
//   | tw | hist [NW][nbins] u32, two images per word (16 bits each) | per-image parameters
// bins per unit of the saturated coordinate y in [0, 1]: y = 1 must still land in bin nbins - 1
__host__ __device__ __forceinline__ float hist_scale(int nbins) { return (float)nbins - 0.015625f; }

template <int TPF>
struct TreeStatsCtx {
    uint32_t* hist;
    const float* sA;        // bin = floor(S * sat(x * A + B)): A = 1 / (histogram range in units of x)
    const float* sScale;    // pixel = x * scale
    const int* sValid;
    float* sBest;           // [warp][NIMG]
    int* sBpos;
    float B, S;             // B = 0.5 (range centred on 0) or 0 (range starts at 0); S = hist_scale(nbins)
    int nbins, nimg;
    bool wide;              // one 32-bit counter per bin and image (N >= 2048) instead of two packed 16-bit ones
};

template <int N>
__device__ __forceinline__ void tree_row_stats(const float (&x)[16], int img, int y, int t, int lane, int warp,
                                               const TreeStatsCtx<N / 16>& cx, float* image_out) {
    constexpr int TPF = N / 16;
    if (!cx.sValid[img]) return;
    const float A = cx.sA[img];
    // 32-bit shared-memory address of this image's histogram, formed once: per pixel one scaled add + one RED
    uint32_t hw = (uint32_t)__cvta_generic_to_shared(cx.hist) + (uint32_t)((cx.wide ? img : (img >> 1)) * cx.nbins) * 4u;
    asm volatile("" : "+r"(hw));          // keep the sum in a register (the compiler re-forms it per pixel otherwise)
    const uint32_t inc = (!cx.wide && (img & 1)) ? 65536u : 1u;
    // bin = floor(S * clamp(x * A + B, 0, 1)) with S = nbins - 2^-6, in two FMA-pipe instructions and no integer
    // clamp: FFMA.SAT maps the histogram range onto [0, 1] (NaN -> 0, +-inf -> the end bins), then one FMA rounded
    // DOWN onto 1.5 * 2^23 (ulp 1) leaves floor(y * S) <= nbins - 1 in the low mantissa bits (no F2I: that runs on
    // the quarter-rate XU pipe).  Per pixel and image: FFMA.SAT, FFMA.RM, LEA, ATOMS and a third of an FMNMX3.
    constexpr int kMagicBits = 0x4B400000;                  // 12582912.0f
    const float S = cx.S;
    hw -= (uint32_t)kMagicBits * 4u;                        // wraps; undone by the scaled add below
    float m = x[0];
#pragma unroll
    for (int e = 0; e < 16; e++) {
        const float yv = __saturatef(fmaf(x[e], A, cx.B));
        const int q = __float_as_int(__fmaf_rd(yv, S, 12582912.0f));
        asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(hw + (uint32_t)q * 4u), "r"(inc) : "memory");
        m = fmaxf(m, x[e]);
    }
    // running peak of this warp: a new maximum is rare after the first rows, so one vote decides.
    // Positions are full row-major indices (a warp may hold two rows when N < 512).
    if (__any_sync(0xffffffffu, m > cx.sBest[warp * cx.nimg + img])) {
        float wm = m;
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) wm = fmaxf(wm, __shfl_xor_sync(0xffffffffu, wm, d));
        int xp = 0x7fffffff;
        if (m == wm) {                   // first element holding the maximum; its position is formed only here
            int eb = 0;
#pragma unroll
            for (int e = 15; e >= 0; e--) if (x[e] == wm) eb = e;
            xp = y * N + t + TPF * eb;
        }
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) xp = min(xp, __shfl_xor_sync(0xffffffffu, xp, d));
        __syncwarp();
        if (lane == 0) { cx.sBest[warp * cx.nimg + img] = wm; cx.sBpos[warp * cx.nimg + img] = xp; }
        __syncwarp();
    }
    if (image_out != nullptr) {
        const float sc = cx.sScale[img];
#pragma unroll
        for (int e = 0; e < 16; e++) image_out[(size_t)y * N + t + TPF * e] = x[e] * sc;
    }
}

// ---- bulk asynchronous copy (TMA, 1-D) completed on an mbarrier: one elected thread moves a whole contiguous
// (row, pair) of the half plane (ncol x 16 bytes) global -> shared; no per-thread copy instructions, no register
// staging, the consumers sleep on the barrier's phase bit (SASS: UBLKCP + SYNCS).
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
// 16-byte asynchronous global -> shared copy (LDGSTS), used where the source is strided (row-pair hand-off)
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(smem_dst)), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int PENDING> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(PENDING) : "memory"); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() {       // make the initialised barriers visible to the async proxy
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void bulk_copy_g2s(void* smem_dst, const void* gsrc, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(smem_dst)), "l"(gsrc), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    uint32_t done;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    } while (!done);
}
// The staging buffer is handed back to the ASYNC proxy (the next bulk copy overwrites it) after a group barrier.  A
// barrier orders generic-proxy accesses among the threads, but the copy engine is another proxy: a shared-memory load
// that has only been ISSUED may still sit in the LSU queue when the elected thread passes the barrier (ptxas sinks the
// instructions that consume the loads past BAR.SYNC), and the engine does not see that queue.  Seen as run-to-run
// differences of 1e-5 in sigma at npix 1024 (two warps per transform), found by searching the same segment twice and
// comparing the records bit for bit (tests: test_repeated_search_is_bit_identical).
// Every reader therefore makes sure its loaded values have ARRIVED before it reaches the barrier: a volatile store of
// a word that depends on every loaded register cannot issue before the loads have returned.  (A cross-proxy fence,
// fence.proxy.async = MEMBAR.ALL.CTA + FENCE.VIEW.ASYNC, is the textbook form; it also drains the histogram atomics
// of the previous transform: +0.7 ms per L-band step.)
__device__ __forceinline__ void loads_arrived_before_release(const float2 (&v)[16], volatile uint32_t* scratch) {
    uint32_t acc = 0u;
#pragma unroll
    for (int e = 0; e < 16; e++) acc |= __float_as_uint(v[e].x);      // .x and .y of an element come from ONE 16-byte load
    *scratch = acc;
}
constexpr int kMaxRowGroups = 32;       // transform groups per row-pass CTA (one mbarrier each)
// entries (16 bytes) of one group's staging buffer in the row pass
template <int N, bool ZM> __host__ __device__ constexpr int row_stage_pitch(int cpad) {
    return ZM ? (cpad > 6 * (N / 16) + 4 ? cpad : 6 * (N / 16) + 4) : cpad;
}

// ------------------------------------------------------------------------------------------
// Tree pass 1, sparse form (N >= 2048 with TB = 2, the row-pair hand-off): the column transform as a PRUNED DFT.  A uv column of the 4096^2 half plane
// holds 32 occupied cells on average out of 4096 (one (baseline, channel) track crosses a column once), so most of a
// column FFT moves and adds zeros.  Split the row index v = 16 m + r (class r = v mod 16) and the output index
// y = k1 + M1 k2 with M1 = N/16:
//     e^{2 pi i v y / N} = e^{2 pi i m k1 / M1} * e^{2 pi i r k1 / N} * e^{2 pi i r k2 / 16},
//     Y_r[k1]       = sum over the cells of class r of  x * e^{2 pi i m k1 / M1}          (direct, occupied cells only)
//     X[k1 + M1 k2] = sum_r (Y_r[k1] W_N^{r k1}) e^{2 pi i r k2 / 16}                      (one radix-16 butterfly)
// One thread owns one k1 of one (column, integration pair): 2 x 16 complex accumulators in registers, the cells
// broadcast from shared memory, the twiddle e^{2 pi i (m k1 mod M1)/M1} from the special-function unit (exact angle).
// No exchange through shared memory, no tile, no scatter; the 16 outputs of a thread are rows k1 + M1 k2 of the
// hand-off, stored straight from registers.
// A CTA keeps ONE column group and walks `spc` consecutive blocks of the launch (consecutive CTAs take the next groups
// for the same blocks, so the 32-byte pieces of a hand-off line are written close together in time while the CTAs stay
// roughly in step; more than ~6 blocks and they drift apart, the lines reach DRAM in pieces and the pass slows down).
// The group's LIST BLOCK, built once per plan by rf_tables.cu, is copied once: the first entry of every (column, class)
// and the entries (m | (cell + 1) << 8) sorted by class, every class padded to an even length with entry 0 = the zero
// cell in front of the values, so the loop takes two cells per turn without a remainder.  The cell values of a block
// (contiguous in the compact grid) arrive by one bulk copy, two turns ahead of the arithmetic.  The warps of a CTA
// never meet at a barrier inside the loop: a buffer is `full` when its copy has landed and `empty` again when all warps
// have arrived after their last read of it (two mbarriers per buffer).
// grid = (ngroups, ceil(n_blk / spc), (TB/2) / NP); block = M1 * NCOL * NP: unit u = tid / M1 = (column u % NCOL, pair u / NCOL).
// Dynamic smem: values [kDftStages][ncmax + 1][TB] float2 (cell 0 of each stays zero) | list block [dft_max_blk] int.
constexpr int kDftStages = 3;         // buffers of k_tree_coldft: the copies run two turns ahead of the arithmetic
__host__ __device__ constexpr int dft_list_header(int ncol) { return (ncol * 16 + 1 + 3) & ~3; }     // ints before the entries

template <int N, int TB, int NCOL, int NP>
__global__ void __launch_bounds__((N / 16) * NCOL * NP) k_tree_coldft(const TreeParams p, const int spc) {
    constexpr int M1 = N / 16, NTH = M1 * NCOL * NP, HDR = dft_list_header(NCOL);
    static_assert(TB == 2, "writes the row-pair hand-off (two lanes fill one 32-byte sector); with the plain layout it loses to the FFTs");
    static_assert(M1 == 256 || M1 == 128, "the low byte of m k1 is the twiddle index");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const size_t xbytes = (size_t)(p.ncmax + 1) * TB * sizeof(float2);
    const int* lblk = reinterpret_cast<const int*>(smem_raw + kDftStages * xbytes);      // the group's list block
    __shared__ __align__(8) uint64_t full[kDftStages], empty[kDftStages], lfull;

    const int tid = threadIdx.x;
    const int g = blockIdx.x, pr0 = blockIdx.z * NP;
    const int s0 = blockIdx.y * spc, ns = min(p.n_blk, s0 + spc) - s0;
    const int c_beg = p.group_cell[g], nc = p.group_cell[g + 1] - c_beg;
    const uint32_t vbytes = (uint32_t)nc * (TB * 8u);
    if (tid < kDftStages) { mbar_init(&full[tid], 1); mbar_init(&empty[tid], NTH / 32); }
    if (tid == kDftStages) mbar_init(&lfull, 1);
    if (tid < kDftStages * (TB / 2))
        reinterpret_cast<float4*>(smem_raw + (size_t)(tid / (TB / 2)) * xbytes)[tid % (TB / 2)] = make_float4(0.f, 0.f, 0.f, 0.f);
    mbar_fence_init();
    __syncthreads();
    // turn n = block s0 + n uses buffer n % kDftStages
    auto fill = [&](int n) {
        const int b = n % kDftStages;
        mbar_arrive_expect_tx(&full[b], vbytes);
        bulk_copy_g2s(smem_raw + (size_t)b * xbytes + TB * 8, p.cellsum + ((size_t)(s0 + n) * p.n_cells + c_beg) * TB, vbytes, &full[b]);
    };
    if (tid == 0) {
        const int off = p.dft_off[g];
        const uint32_t lb = (uint32_t)(p.dft_off[g + 1] - off) * 4u;
        mbar_arrive_expect_tx(&lfull, lb);
        bulk_copy_g2s(smem_raw + kDftStages * xbytes, p.dft_blk + off, lb, &lfull);
        if (nc > 0)
            for (int n = 0; n < kDftStages - 1 && n < ns; n++) fill(n);
    }

    const int u = tid / M1, k1 = tid % M1;
    const int c = u % NCOL, pp = u / NCOL, pr = pr0 + pp;
    const float2 w1 = __ldg(p.twiddles + 16 + k1);         // exp(2 pi i k1 / N), k1 < 256
    const float sc = p.norm;
    const int col = g * NCOL + c;
    const bool col0 = col == 0;
    mbar_wait(&lfull, 0);
    const int* ucls = lblk + c * 16;
    const int* lst = lblk + HDR;
    for (int n = 0; n < ns; n++) {
        const int buf = n % kDftStages;
        float4* Hs = reinterpret_cast<float4*>(p.Ht + (size_t)(s0 + n) * N * p.cpad * TB);
        if (nc > 0 && tid == 0 && n + kDftStages - 1 < ns) {
            // the buffer of turn n + kDftStages - 1 is the one turn n - 1 read: every warp has arrived on `empty` after its
            // last read (a fresh barrier passes the wait for parity 1, so the first fill of a buffer does not block)
            const int k = n + kDftStages - 1;
            mbar_wait(&empty[k % kDftStages], ((k / kDftStages) & 1) ^ 1);
            fill(k);
        }
        if (nc > 0) mbar_wait(&full[buf], (n / kDftStages) & 1);
        const float4* ux = reinterpret_cast<const float4*>(smem_raw + (size_t)buf * xbytes) + pr;   // cell 0 = zeros, cell i + 1 = cell i of the group
        auto x_of = [&](int e) { return ux[(e >> 8) * (TB / 2)]; };
        // e^{2 pi i (m k1 mod M1) / M1}: the angle is an exact multiple of 2 pi / M1 below 2 pi, so the two special-function
        // evaluations are good to ~5e-7 absolute (an M1-entry table in shared memory costs 3.5 wavefronts per read: the
        // stride m k1 of a warp's 32 consecutive k1 conflicts for every m that is not odd)
        auto tw_of = [&](int e) {
            // j as a float without the conversion unit (it shares the special-function pipe): 2^23 + j is exact
            const uint32_t prod = (uint32_t)(e * k1) & (M1 == 256 ? 0xffffffffu : 0xffffff7fu);
            const float fj = __uint_as_float(__byte_perm(prod, 0x4B000000u, 0x7650));      // low byte of prod under 0x4B0000..
            constexpr float kStep = 6.283185307179586f / (float)M1;
            const float a = fmaf(fj, kStep, -8388608.f * kStep);
            float2 w;
            __sincosf(a, &w.y, &w.x);
            return w;
        };
        float2 ya[16], yb[16];
#pragma unroll
        for (int r = 0; r < 16; r++) { ya[r] = make_float2(0.f, 0.f); yb[r] = make_float2(0.f, 0.f); }
        {
            int i = ucls[0];
            int e0 = lst[i], e1 = lst[i + 1];
            float4 x0 = x_of(e0), x1 = x_of(e1);
            float2 w0 = tw_of(e0), w1c = tw_of(e1);
#pragma unroll
            for (int r = 0; r < 16; r++) {
                const int end = ucls[r + 1];
#pragma unroll 1
                while (i < end) {                 // two cells per turn; the list is padded, the classes are even
                    e0 = lst[i + 2];
                    e1 = lst[i + 3];
                    ya[r].x = fmaf(x0.x, w0.x, ya[r].x); ya[r].x = fmaf(-x0.y, w0.y, ya[r].x);
                    ya[r].y = fmaf(x0.x, w0.y, ya[r].y); ya[r].y = fmaf(x0.y, w0.x, ya[r].y);
                    yb[r].x = fmaf(x0.z, w0.x, yb[r].x); yb[r].x = fmaf(-x0.w, w0.y, yb[r].x);
                    yb[r].y = fmaf(x0.z, w0.y, yb[r].y); yb[r].y = fmaf(x0.w, w0.x, yb[r].y);
                    ya[r].x = fmaf(x1.x, w1c.x, ya[r].x); ya[r].x = fmaf(-x1.y, w1c.y, ya[r].x);
                    ya[r].y = fmaf(x1.x, w1c.y, ya[r].y); ya[r].y = fmaf(x1.y, w1c.x, ya[r].y);
                    yb[r].x = fmaf(x1.z, w1c.x, yb[r].x); yb[r].x = fmaf(-x1.w, w1c.y, yb[r].x);
                    yb[r].y = fmaf(x1.z, w1c.y, yb[r].y); yb[r].y = fmaf(x1.w, w1c.x, yb[r].y);
                    x0 = x_of(e0); w0 = tw_of(e0);
                    x1 = x_of(e1); w1c = tw_of(e1);
                    i += 2;
                }
            }
        }
        // the values of this turn are consumed: hand the buffer back (the loads fed the multiply-adds above, so they have
        // arrived; the read-ahead past the list points at the zero cell, which no copy writes)
        __syncwarp();
        if (nc > 0 && (tid & 31) == 0) mbar_arrive(&empty[buf]);
        // ---- twiddles W_N^{r k1} (with the normalisation folded in), radix-16 butterfly over the classes
        {
            float2 w[16];
            w[1] = w1;
#pragma unroll
            for (int t = 2; t < 16; t++) w[t] = (t & 1) ? cmul(w[t - 1], w1) : cmul(w[t / 2], w[t / 2]);
            ya[0] = make_float2(ya[0].x * sc, ya[0].y * sc);
            yb[0] = make_float2(yb[0].x * sc, yb[0].y * sc);
#pragma unroll
            for (int t = 1; t < 16; t++) {
                const float2 ws = make_float2(w[t].x * sc, w[t].y * sc);
                ya[t] = cmul(ya[t], ws);
                yb[t] = cmul(yb[t], ws);
            }
        }
        bfly<16>(ya);
        bfly<16>(yb);
        // ---- store rows k1 + M1 k2 of H (row-pair layout of k_tree_colfft<..., RP>); streaming: the row pass reads them a whole launch later
        {
#pragma unroll
            for (int k2 = 0; k2 < 16; k2++) {
                const int y = k1 + M1 * k2;
                float4 o = make_float4(ya[k2].x, ya[k2].y, yb[k2].x, yb[k2].y);
                if (col0) { o.y = 0.f; o.w = 0.f; }       // column 0 is Hermitian along v: its transform is real (B2)
                __stcs(&Hs[(((size_t)(y >> 1)) * (TB / 2) + pr) * p.cpad * 2 + rp_entry(col, y & 1)], o);
            }
        }
    }
}

constexpr int kThreads2 = 512;          // tree pass 2: one CTA of 16 warps per SM
constexpr int kWarps2 = kThreads2 / 32;

// NT2 = threads per CTA: 512 (one CTA per SM) up to N = 1024; 256 for N >= 2048, where one transform already
// needs 128 or 256 threads and two or three smaller CTAs per SM hide its barriers better than one large one.
// ZM: the half plane occupies at most 6 N/16 columns (ncol <= 6 TPF; always true with the default cell, A13), so
// elements 6 TPF .. 10 TPF - 1 of every row spectrum are zero: not staged into registers, pruned from the first stage.
// RP: the hand-off has the row-pair layout of k_tree_colfft<..., RP = true> (TB = 2): one bulk copy stages a DOUBLE
// row (ncol x 32 bytes, entries rp_entry(c, y & 1)).  The group unpacks BOTH rows into registers at once and hands the
// buffer back, so the next double row is copied behind two row transforms.
template <int N, int TB, int NT2, bool ZM, bool RP = false>
__global__ void __launch_bounds__(NT2, N >= 2048 ? 2 : 1) k_tree_rowfft_stats(const TreeParams p) {
    static_assert(!RP || TB == 2, "the row-pair hand-off holds one pair per row");
    constexpr int RPH = RP ? 2 : 1;                   // rows per staged item
    constexpr bool PADDED = ZM && !RP;                // staging buffer zero-padded to 6 TPF columns: unconditional loads
    constexpr int NWP = NT2 / 32;
    using C = FftCfg<N>;
    constexpr int G2 = NT2 / C::TPF;
    constexpr int XB = fft_padded_size(N);
    constexpr int NIMG = 2 * TB - 1;
    constexpr bool WIDE = N >= 2048;                  // 16-bit counters would wrap: N^2 pixels in few central bins
    constexpr int NW = WIDE ? NIMG : (NIMG + 1) / 2;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2* xbuf = reinterpret_cast<float2*>(smem_raw);
    // region 0 holds the FFT exchange buffers, later the unpacked histogram + prefix sums
    const int region0 = max(G2 * XB, p.nbins);                               // float2 units
    float2* tw = xbuf + region0;
    float2* twp = tw + C::TW_TOTAL;                                          // [16][15] stage-2 twiddle powers
    // staged (row, pair) of each group, [G2][sgp]: ZM reads columns 0 .. 6 TPF unconditionally, so the buffer spans them
    // and everything past ncol stays zero (the bulk copy writes ncol entries only)
    const int sgp = RPH * row_stage_pitch<N, PADDED>(p.cpad);     // entries of one staged item
    float4* stg = reinterpret_cast<float4*>(twp + kTwpSize);
    uint32_t* hist = reinterpret_cast<uint32_t*>(stg + (size_t)G2 * sgp);    // [NW][nbins]
    float* sA = reinterpret_cast<float*>(hist + (size_t)NW * p.nbins);       // [16]
    float* sScale = sA + 16;                                                 // [16]
    float* sSig = sScale + 16;                                               // [16] sigma_rms per image
    int* sValid = reinterpret_cast<int*>(sSig + 16);                         // [16]
    int* sInr = sValid + 16;                                                 // [16] 1 = an image of the search loop
    float* sBest = reinterpret_cast<float*>(sInr + 16);                      // [16 warps][NIMG]
    int* sBpos = reinterpret_cast<int*>(sBest + NWP * NIMG);             // [16 warps][NIMG]
    uint32_t* hun = reinterpret_cast<uint32_t*>(xbuf);                       // after the row loop
    uint32_t* cum = hun + p.nbins;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int slot = blockIdx.x;
    const BlockDesc blk = p.blocks[slot];
    if (blk.tb * TB >= blk.nsearch) return;          // padding block of a gather group: no image (uniform for the CTA)
    const float2* Hblk = p.Ht + (size_t)slot * N * p.cpad * TB;
    const int grp = tid / C::TPF, t = tid % C::TPF;
    float4* sg = stg + (size_t)grp * sgp;

    __shared__ __align__(8) uint64_t mbar[kMaxRowGroups];
    __shared__ uint32_t rel_scratch[32];       // see loads_arrived_before_release
    // Staging: (row y, pair p2) = ncol contiguous 16-byte (H_a, H_b) entries = ONE bulk copy issued by the group's first
    // thread.  The group walks rows grp, grp + G2, ... and the TB/2 pairs of each, so the source advances by one
    // (row, pair) inside a row and by (G2 - 1) TB/2 + 1 of them at the end of a row: a running pointer, no index math.
    // (RP: an item is a double row of cpad x 32 bytes, one pair per row)
    const char* src_next = reinterpret_cast<const char*>(Hblk) + (size_t)grp * (TB / 2) * p.cpad * (16 * RPH);
    const uint32_t copy_bytes = (uint32_t)p.ncol * (16u * RPH);
    const size_t step_pair = (size_t)p.cpad * (16 * RPH), step_row = ((size_t)(G2 - 1) * (TB / 2) + 1) * p.cpad * (16 * RPH);
    auto stage_next = [&](bool end_of_row) {
        if (t == 0) {
            mbar_arrive_expect_tx(&mbar[grp], copy_bytes);
            bulk_copy_g2s(sg, src_next, copy_bytes, &mbar[grp]);
        }
        src_next += end_of_row ? step_row : step_pair;
    };
    for (int i = tid; i < G2 * sgp; i += NT2) stg[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    if (tid < kMaxRowGroups) mbar_init(&mbar[tid], 1);
    mbar_fence_init();                   // also orders the zero fill (generic proxy) before the first bulk copy
    __syncthreads();
    stage_next(TB == 2);
    uint32_t phase = 0;

    for (int i = tid; i < NW * p.nbins; i += NT2) hist[i] = 0u;
    load_twiddles<N>(tw, p.twiddles, tid, NT2);
    for (int i = tid; i < kTwpSize; i += NT2) twp[i] = p.twp[i];
    for (int i = tid; i < NWP * NIMG; i += NT2) { sBest[i] = -CUDART_INF_F; sBpos[i] = 0; }
    if (tid < NIMG) {
        int l = 0, off = 0;
        while (tid >= off + (TB >> l)) { off += TB >> l; l++; }
        const int i = tid - off, dt = 1 << l;
        const int j = blk.tb * (TB >> l) + i;
        float tot = 0.f;
        for (int part = 0; part < p.n_parts; part++) tot += p.sumsq[((size_t)slot * NIMG + tid) * p.n_parts + part];
        const float sig = sqrtf(tot) / (float)dt;                // rms of the image (Parseval)
        const bool inr = p.dt_idx[l] >= 0 && (j + 1) * dt <= blk.nsearch;
        const bool valid = inr && sig > 0.f;              // an all-zero image has snr := 0 and is never a candidate
        sInr[tid] = inr ? 1 : 0;
        sValid[tid] = valid ? 1 : 0;
        sSig[tid] = sig;
        sScale[tid] = 1.f / (float)dt;
        sA[tid] = valid ? 1.f / (2.f * kHistRange * sig) / (float)dt : 0.f;     // x is the SUM of dt integrations
    }
    __syncthreads();

    TreeStatsCtx<C::TPF> cx{hist, sA, sScale, sValid, sBest, sBpos, 0.5f, hist_scale(p.nbins), p.nbins, NIMG, WIDE};
    float2* xb = xbuf + grp * XB;
    const bool dbg = p.image_out != nullptr && slot == p.dbg_slot;

    // unpack one staged row into the transform input: Z[c] = H_a[c] + i H_b[c], Z[N - c] = conj(H_a[c]) + i conj(H_b[c]);
    // the column pass stores exact zeros in the imaginary parts of column 0 (rounding noise of a Hermitian column, B2)
    auto unpack = [&](float2 (&v)[16], int hrow) {
#pragma unroll
        for (int e = 0; e < 16; e++) {
            if (ZM && e >= 6 && e <= 9) { v[e] = make_float2(0.f, 0.f); continue; }
            if (PADDED) {
                const float4 hv = sg[(e < 8) ? t + C::TPF * e : N - C::TPF * e - t];   // past ncol: zeros
                v[e] = (e < 8) ? make_float2(hv.x - hv.w, hv.y + hv.z) : make_float2(hv.x + hv.w, hv.z - hv.y);
            } else {
                const int c = t + C::TPF * e;
                const int cc = (e < 8) ? c : N - c;
                float4 hv = make_float4(0.f, 0.f, 0.f, 0.f);
                if (cc < p.ncol) hv = sg[RP ? rp_entry(cc, hrow) : cc];
                if (cc == 0 || cc == N / 2) v[e] = make_float2(hv.x, hv.z);
                else if (e < 8) v[e] = make_float2(hv.x - hv.w, hv.y + hv.z);
                else v[e] = make_float2(hv.x + hv.w, hv.z - hv.y);
            }
        }
    };
    for (int yb = grp * RPH; yb < N; yb += G2 * RPH) {
      float2 vB[RP ? 16 : 1];                         // RP: the second row of the double row, held while the first is transformed
#pragma unroll 1
      for (int h = 0; h < RPH; h++) {
        const int y = yb + h;
        float s2p[16], s4p[16];
#pragma unroll 1
        for (int p2 = 0; p2 < TB / 2; p2++) {
            float2 v[16];
            if (!RP || h == 0) {
                mbar_wait(&mbar[grp], phase);                    // the (row, pair) [RP: the double row] has landed
                phase ^= 1u;
                unpack(v, 0);
                loads_arrived_before_release(v, &rel_scratch[warp]);
                if constexpr (RP) {
                    unpack(vB, 1);
                    loads_arrived_before_release(vB, &rel_scratch[warp]);
                }
                fft_group_sync<C::TPF>(1 + grp);                 // staging buffer consumed
                // prefetch the next (row, pair) of this group while this one is transformed
                const bool last_pair = p2 + 1 == TB / 2;
                if (RP) { if (yb + G2 * RPH < N) stage_next(true); }
                else if (!last_pair || y + G2 < N) stage_next(p2 + 2 == TB / 2 || (TB == 2));
            } else {
                if constexpr (RP) {
#pragma unroll
                    for (int e = 0; e < 16; e++) v[e] = vB[e];
                }
            }
            fft_inverse<N, ZM, (N >= 2048)>(v, xb, tw, t, 1 + grp, twp);
            float a[16], s2[16];
#pragma unroll
            for (int e = 0; e < 16; e++) a[e] = v[e].x;
            tree_row_stats<N>(a, 2 * p2, y, t, lane, warp, cx, (dbg && p.dbg_img == 2 * p2) ? p.image_out : nullptr);
#pragma unroll
            for (int e = 0; e < 16; e++) { a[e] = v[e].y; s2[e] = v[e].x + v[e].y; }
            tree_row_stats<N>(a, 2 * p2 + 1, y, t, lane, warp, cx, (dbg && p.dbg_img == 2 * p2 + 1) ? p.image_out : nullptr);
            {
                const int img = TB + p2;
                tree_row_stats<N>(s2, img, y, t, lane, warp, cx, (dbg && p.dbg_img == img) ? p.image_out : nullptr);
            }
            if (TB >= 4) {
                if (p2 & 1) {
                    float s4[16];
#pragma unroll
                    for (int e = 0; e < 16; e++) s4[e] = s2p[e] + s2[e];
                    const int img = TB + TB / 2 + (p2 >> 1);
                    tree_row_stats<N>(s4, img, y, t, lane, warp, cx, (dbg && p.dbg_img == img) ? p.image_out : nullptr);
                    if (TB >= 8) {
                        if (p2 == 3) {
#pragma unroll
                            for (int e = 0; e < 16; e++) s4[e] += s4p[e];
                            const int img8 = TB + TB / 2 + TB / 4;
                            tree_row_stats<N>(s4, img8, y, t, lane, warp, cx, (dbg && p.dbg_img == img8) ? p.image_out : nullptr);
                        } else {
#pragma unroll
                            for (int e = 0; e < 16; e++) s4p[e] = s4[e];
                        }
                    }
                } else {
#pragma unroll
                    for (int e = 0; e < 16; e++) s2p[e] = s2[e];
                }
            }
        }
      }
    }
    __syncthreads();

    // ---- per image: unpack the histogram, prefix sums, median / MAD, S/N, threshold
    for (int img = 0; img < NIMG; img++) {
        const bool report_zero = p.stats_out != nullptr && slot == p.dbg_slot && img == p.dbg_img;
        if (!sValid[img] && !report_zero) continue;            // block-uniform
        const uint32_t* hw = hist + (WIDE ? img : (img >> 1)) * p.nbins;
        const int sh = WIDE ? 0 : (img & 1) * 16;
        const int per = (p.nbins + NT2 - 1) / NT2;                 // bins [tid * per, ...) of this thread (none past nbins)
        const int nmine = max(0, min(per, p.nbins - tid * per));
        uint32_t local = 0;
        for (int i = 0; i < nmine; i++) {
            const uint32_t c = WIDE ? hw[tid * per + i] : (hw[tid * per + i] >> sh) & 0xffffu;
            hun[tid * per + i] = c;
            local += c;
        }
        uint32_t inc = local;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            uint32_t o = __shfl_up_sync(0xffffffffu, inc, d);
            if (lane >= d) inc += o;
        }
        __shared__ uint32_t wtot[NWP];
        if (lane == 31) wtot[warp] = inc;
        __syncthreads();
        uint32_t base = inc - local, total = 0;
        for (int w = 0; w < NWP; w++) { if (w < warp) base += wtot[w]; total += wtot[w]; }
        for (int i = 0; i < nmine; i++) { cum[tid * per + i] = base; base += hun[tid * per + i]; }
        __syncthreads();
        if (warp == 0) {
            int overflow = 0;
            float sigma = 0.f;
            const float sig_rms = sSig[img];
            if (sValid[img]) {
                if (total != (uint32_t)N * (uint32_t)N) overflow = 1;   // a 16-bit counter wrapped
                HistView hv{hun, cum, p.nbins, -kHistRange * sig_rms, hist_scale(p.nbins) / (2.f * kHistRange * sig_rms)};
                sigma = robust_sigma_from_hist(hv, (float)N * (float)N, lane, &overflow);
            }
            if (lane == 0) {
                float bv = -CUDART_INF_F;
                int bp = 0;
                for (int w = 0; w < NWP; w++) {
                    const float ov = sBest[w * NIMG + img];
                    const int op = sBpos[w * NIMG + img];
                    if (ov > bv || (ov == bv && op < bp)) { bv = ov; bp = op; }
                }
                int l = 0, off = 0;
                while (img >= off + (TB >> l)) { off += TB >> l; l++; }
                const float peak = sValid[img] ? bv * sScale[img] : 0.f;
                const float snr = sigma > 0.f ? peak / sigma : 0.f;
                const int x = bp % N, yy = bp / N;
                rf_cand c;
                c.dm_idx = blk.dm_idx; c.dt_idx = p.dt_idx[l]; c.t_idx = blk.tb * (TB >> l) + (img - off);
                c.l_pix = x < N / 2 ? x : x - N;
                c.m_pix = yy < N / 2 ? yy : yy - N;
                c.peak = peak; c.sigma = sigma; c.snr = snr;
                if (overflow) atomicAdd(&p.counters[0], 1);
                if (report_zero) *p.stats_out = c;
                if (p.cand_count != nullptr && sValid[img] && sigma > 0.f && snr >= p.threshold) {
                    int idx = atomicAdd(p.cand_count, 1);
                    if (idx < p.cand_capacity) p.cand_items[idx] = c;
                }
            }
        }
        __syncthreads();
    }
    // images of the search loop this CTA has finalised (rf_counters.images is counted on the device)
    if (tid == 0 && p.cand_count != nullptr) {
        int n = 0;
        for (int img = 0; img < NIMG; img++) n += sInr[img];
        if (n) atomicAdd(&p.counters[1], n);
    }
}

// ==========================================================================================
// Periodicity search ("reading a time segment, transforming it to frequencies with a
// Fourier transform, and imaging each frequency", PAPER.md:100 footnote 4; reading A23).
//
// k_time_fft<NT>: for one DM trial, S[k] = (1/NT) sum_t s[t] e^{-2 pi i k t/NT} of the dedispersed Stokes-I
// series of every (baseline, channel), written for k = 1..NT/2 as the PAIR (S[k], -i S[k]) at
// "integrations" 2(k-1), 2(k-1)+1 of a visI-shaped slab.  Hermitian imaging of S gives Re I_k and of -i S
// gives Im I_k (I_k = the complex image of S[k]), so the unchanged gather / column-FFT kernels and the pair
// transform of the row pass deliver the complex image of every fluctuation frequency.
// grid = ceil(nelem / G) with G = 256 / (NT/16) transforms per CTA; smem: G exchange buffers | twiddles.
template <int NT>
__global__ void __launch_bounds__(kThreads) k_time_fft(const float2* __restrict__ visI, const int32_t* __restrict__ delay_dm,
                                                       const float2* __restrict__ twiddles, float2* __restrict__ slab,
                                                       int nelem, int nchan, int tpitch_in, int tpitch_out) {
    using C = FftCfg<NT>;
    constexpr int G = kThreads / C::TPF;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2* xbuf = reinterpret_cast<float2*>(smem_raw);
    float2* tw = xbuf + G * fft_padded_size(NT);
    const int tid = threadIdx.x, grp = tid / C::TPF, t = tid % C::TPF;
    load_twiddles<NT>(tw, twiddles, tid, kThreads);
    __syncthreads();
    const int e = blockIdx.x * G + grp;
    const bool live = e < nelem;
    const int ee = live ? e : nelem - 1;             // idle groups repeat the last element (barriers stay uniform)
    const float2* src = visI + (size_t)ee * tpitch_in + delay_dm[ee % nchan];
    float2 v[16];
#pragma unroll
    for (int k = 0; k < 16; k++) { const float2 x = __ldg(src + t + C::TPF * k); v[k] = make_float2(x.x, -x.y); }
    fft_inverse<NT>(v, xbuf + grp * fft_padded_size(NT), tw, t, 1 + grp);     // forward = conj(inverse(conj))
    if (!live) return;
    const float sc = 1.f / (float)NT;
    float4* dst = reinterpret_cast<float4*>(slab + (size_t)e * tpitch_out);
#pragma unroll
    for (int k = 0; k < 16; k++) {
        const int kk = t + C::TPF * k;                // natural order: fluctuation-frequency bin
        if (kk >= 1 && kk <= NT / 2) {
            const float re = v[k].x * sc, im = -v[k].y * sc;
            dst[kk - 1] = make_float4(re, im, im, -re);          // (S, -i S)
        }
    }
}

// Row pass of the periodicity search.  Same structure as k_tree_rowfft_stats (one CTA per block, staged
// (row, pair) input, pair transform), but each pair IS one image: a = Re I_k, b = Im I_k, searched in power
// P = a^2 + b^2.  Histogram over [0, kPowerRange * mean P] (mean P from Parseval), median by interpolation,
// sigma = sqrt(median / ln 2), snr = sqrt(peak) / sigma.  Candidate: dt_idx = -1, t_idx = k.
constexpr float kPowerRange = 6.f;

template <int N, int TB>
__global__ void __launch_bounds__(kThreads2, 1) k_tree_rowfft_power(const TreeParams p) {
    using C = FftCfg<N>;
    constexpr int G2 = kThreads2 / C::TPF;
    constexpr int XB = fft_padded_size(N);
    constexpr int NIMG = TB / 2;                      // one power image per pair
    constexpr int NNODE = 2 * TB - 1;                 // Parseval nodes written by the gather kernel
    constexpr int NSL = 2 * NIMG;                     // image i uses statistics slot 2 i: a whole 32-bit counter per bin
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2* xbuf = reinterpret_cast<float2*>(smem_raw);
    const int region0 = max(G2 * XB, p.nbins);
    float2* tw = xbuf + region0;
    float4* stg = reinterpret_cast<float4*>(tw + C::TW_TOTAL);
    uint32_t* hist = reinterpret_cast<uint32_t*>(stg + (size_t)G2 * p.cpad);   // [NIMG][nbins]
    float* sA = reinterpret_cast<float*>(hist + (size_t)NIMG * p.nbins);
    float* sScale = sA + 16;
    float* sMean = sScale + 16;                       // mean power per image (Parseval)
    int* sValid = reinterpret_cast<int*>(sMean + 16);
    float* sBest = reinterpret_cast<float*>(sValid + 16);
    int* sBpos = reinterpret_cast<int*>(sBest + kWarps2 * NSL);
    uint32_t* hun = reinterpret_cast<uint32_t*>(xbuf);
    uint32_t* cum = hun + p.nbins;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int slot = blockIdx.x;
    const BlockDesc blk = p.blocks[slot];
    const float2* Hblk = p.Ht + (size_t)slot * N * p.cpad * TB;
    const int grp = tid / C::TPF, t = tid % C::TPF;
    float4* sg = stg + (size_t)grp * p.cpad;
    __shared__ __align__(8) uint64_t mbar[kMaxRowGroups];
    __shared__ uint32_t rel_scratch[32];       // see loads_arrived_before_release
    auto stage = [&](int y, int p2) {
        const float4* src = reinterpret_cast<const float4*>(Hblk + ((size_t)y * (TB / 2) + p2) * p.cpad * 2);
        if (t == 0) {
            mbar_arrive_expect_tx(&mbar[grp], (uint32_t)p.ncol * 16u);
            bulk_copy_g2s(sg, src, (uint32_t)p.ncol * 16u, &mbar[grp]);
        }
    };
    if (tid < kMaxRowGroups) mbar_init(&mbar[tid], 1);
    mbar_fence_init();
    __syncthreads();
    stage(grp, 0);
    uint32_t phase = 0;
    for (int i = tid; i < NIMG * p.nbins; i += kThreads2) hist[i] = 0u;
    load_twiddles<N>(tw, p.twiddles, tid, kThreads2);
    for (int i = tid; i < kWarps2 * NSL; i += kThreads2) { sBest[i] = -CUDART_INF_F; sBpos[i] = 0; }
    if (tid < 16) { sValid[tid] = 0; sA[tid] = 0.f; sScale[tid] = 1.f; sMean[tid] = 0.f; }
    __syncthreads();
    if (tid < NIMG) {
        float tot = 0.f;                               // mean P = mean(a^2) + mean(b^2): level-0 nodes 2i, 2i+1
        for (int h = 0; h < 2; h++)
            for (int part = 0; part < p.n_parts; part++) tot += p.sumsq[((size_t)slot * NNODE + 2 * tid + h) * p.n_parts + part];
        const int k = 1 + blk.tb * NIMG + tid;         // fluctuation-frequency bin of this image
        const bool valid = k <= blk.nsearch / 2 && tot > 0.f;      // nsearch = NT of this DM
        if (k <= blk.nsearch / 2 && p.cand_count != nullptr) atomicAdd(&p.counters[1], 1);   // frequency images searched
        sValid[2 * tid] = valid ? 1 : 0;
        sMean[2 * tid] = tot;
        sA[2 * tid] = valid ? 1.f / (kPowerRange * tot) : 0.f;
    }
    __syncthreads();

    TreeStatsCtx<C::TPF> cx{hist, sA, sScale, sValid, sBest, sBpos, 0.f, hist_scale(p.nbins), p.nbins, NSL, false};
    float2* xb = xbuf + grp * XB;
    const bool dbg = p.image_out != nullptr && slot == p.dbg_slot;
    for (int y = grp; y < N; y += G2) {
#pragma unroll 1
        for (int p2 = 0; p2 < TB / 2; p2++) {
            float2 v[16];
            mbar_wait(&mbar[grp], phase);
            phase ^= 1u;
#pragma unroll
            for (int e = 0; e < 16; e++) {
                const int c = t + C::TPF * e;
                const int cc = (e < 8) ? c : N - c;
                float4 h = make_float4(0.f, 0.f, 0.f, 0.f);
                if (cc < p.ncol) h = sg[cc];
                if (cc == 0 || cc == N / 2) v[e] = make_float2(h.x, h.z);
                else if (e < 8) v[e] = make_float2(h.x - h.w, h.y + h.z);
                else v[e] = make_float2(h.x + h.w, h.z - h.y);
            }
            loads_arrived_before_release(v, &rel_scratch[warp]);
            fft_group_sync<C::TPF>(1 + grp);
            {
                const int np2 = (p2 + 1 == TB / 2) ? 0 : p2 + 1;
                const int ny = (p2 + 1 == TB / 2) ? y + G2 : y;
                if (ny < N) stage(ny, np2);
            }
            fft_inverse<N>(v, xb, tw, t, 1 + grp);
            float pw[16];
#pragma unroll
            for (int e = 0; e < 16; e++) pw[e] = fmaf(v[e].x, v[e].x, v[e].y * v[e].y);
            tree_row_stats<N>(pw, 2 * p2, y, t, lane, warp, cx, (dbg && p.dbg_img == p2) ? p.image_out : nullptr);
        }
    }
    __syncthreads();

    for (int img = 0; img < NIMG; img++) {
        const int si = 2 * img;
        const bool report_zero = p.stats_out != nullptr && slot == p.dbg_slot && img == p.dbg_img;
        if (!sValid[si] && !report_zero) continue;
        const uint32_t* hw = hist + (size_t)img * p.nbins;
        const int per = p.nbins / kThreads2;
        uint32_t local = 0;
        for (int i = 0; i < per; i++) {
            const uint32_t c = hw[tid * per + i];
            hun[tid * per + i] = c;
            local += c;
        }
        uint32_t inc = local;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            uint32_t o = __shfl_up_sync(0xffffffffu, inc, d);
            if (lane >= d) inc += o;
        }
        __shared__ uint32_t wtot[kWarps2];
        if (lane == 31) wtot[warp] = inc;
        __syncthreads();
        uint32_t base = inc - local;
        for (int w = 0; w < warp; w++) base += wtot[w];
        for (int i = 0; i < per; i++) { cum[tid * per + i] = base; base += hun[tid * per + i]; }
        __syncthreads();
        if (tid == 0) {
            int overflow = 0;
            float sigma = 0.f;
            if (sValid[si]) {
                // median: the bin where the cumulative count crosses N^2/2, linear inside the bin
                const float target = 0.5f * (float)N * (float)N;
                int lo_b = 0, hi_b = p.nbins - 1;
                while (lo_b < hi_b) {
                    const int mid = (lo_b + hi_b + 1) >> 1;
                    if ((float)cum[mid] <= target) lo_b = mid; else hi_b = mid - 1;
                }
                const float hb = (float)hun[lo_b];
                const float w = kPowerRange * sMean[si] / hist_scale(p.nbins);
                const float med = ((float)lo_b + (hb > 0.f ? (target - (float)cum[lo_b]) / hb : 0.5f)) * w;
                if (lo_b == p.nbins - 1) overflow = 1;           // median beyond the histogram range
                sigma = sqrtf(med / 0.6931471805599453f);
            }
            float bv = -CUDART_INF_F;
            int bp = 0;
            for (int w = 0; w < kWarps2; w++) {
                const float ov = sBest[w * NSL + si];
                const int op = sBpos[w * NSL + si];
                if (ov > bv || (ov == bv && op < bp)) { bv = ov; bp = op; }
            }
            const float peak = sValid[si] ? sqrtf(fmaxf(bv, 0.f)) : 0.f;
            const float snr = sigma > 0.f ? peak / sigma : 0.f;
            const int x = bp % N, yy = bp / N;
            rf_cand c;
            c.dm_idx = blk.dm_idx; c.dt_idx = -1; c.t_idx = 1 + blk.tb * NIMG + img;
            c.l_pix = x < N / 2 ? x : x - N;
            c.m_pix = yy < N / 2 ? yy : yy - N;
            c.peak = peak; c.sigma = sigma; c.snr = snr;
            if (overflow) atomicAdd(&p.counters[0], 1);
            if (report_zero) *p.stats_out = c;
            if (p.cand_count != nullptr && sValid[si] && sigma > 0.f && snr >= p.threshold) {
                int idx = atomicAdd(p.cand_count, 1);
                if (idx < p.cand_capacity) p.cand_items[idx] = c;
            }
        }
        __syncthreads();
    }
}

}  // namespace rf
