// rf_search.cu -- workspace, kernel dispatch and the batch loop of rf_search.
//
// The search loop over (DM trial x sampling time x integration) (Fig. 2) is
// flattened at plan time into device-resident work lists (blocks of the boxcar-tree path, images of the
// per-image path); rf_search walks them in batches sized to whole waves of row-pass CTAs within a
// workspace budget for the half-plane hand-off between the two FFT passes.
#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <cstring>

#include "rf_tree_kernels.cuh"

namespace rf {

// Kernel attributes are per-device state: every plan (created on one device, rf_plan::device) opts each kernel into
// its dynamic shared memory itself, once per size increase.  Requests at or below the 48 KB default need no opt-in.
int ensure_smem_attr(rf_plan* p, const void* kern, size_t smem) {
    if (smem <= 48 * 1024) return RF_OK;
    if (smem > kMaxDynSmem) { set_error("internal: kernel needs %zu bytes of shared memory (limit %zu)", smem, kMaxDynSmem); return RF_ERR_STATE; }
    size_t& have = p->smem_attr[kern];
    if (smem <= have) return RF_OK;
    RF_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    have = smem;
    return RF_OK;
}

namespace {

template <int N> size_t smem_pass1(int nchan, int ncolgrp) {
    return (size_t)ncolgrp * (fft_padded_size(N) + 1) * sizeof(float2) +
           FftCfg<N>::TW_TOTAL * sizeof(float2) + (size_t)nchan * sizeof(int) + 8 * sizeof(float);
}
template <int N> constexpr bool exact_stats() { return N <= 128; }
template <int N> size_t smem_pass2(int nbins) {
    return (size_t)(kThreads / FftCfg<N>::TPF) * fft_padded_size(N) * sizeof(float2) +
           FftCfg<N>::TW_TOTAL * sizeof(float2) + (size_t)3 * nbins * sizeof(uint32_t) +
           (16 + 16 + 8 + 4) * 4 + (exact_stats<N>() ? (size_t)2 * N * N * sizeof(float) : 0);
}

template <int N, int NPOL, int NCOL>
int launch_pass1(rf_plan* p, const SearchParams& sp, int nchan, cudaStream_t st) {
    auto kern = k_grid_colfft<N, NPOL, NCOL>;
    const size_t smem = smem_pass1<N>(nchan, NCOL);
    { const int rc_a = ensure_smem_attr(p, (const void*)kern, smem); if (rc_a != RF_OK) return rc_a; }
    kern<<<dim3(sp.n_img, sp.ngroups), kThreads, smem, st>>>(sp);
    RF_CUDA_CHECK(cudaGetLastError());
    return RF_OK;
}

template <int N, int NCOL>
int launch_pass1_npol(rf_plan* p, const SearchParams& sp, int nchan, int npol, cudaStream_t st) {
    switch (npol) {
        case 1: return launch_pass1<N, 1, NCOL>(p, sp, nchan, st);
        case 2: return launch_pass1<N, 2, NCOL>(p, sp, nchan, st);
        case 4: return launch_pass1<N, 4, NCOL>(p, sp, nchan, st);
    }
    set_error("unsupported npol %d", npol);
    return RF_ERR_ARG;
}

template <int N>
int launch_pass2(rf_plan* p, const SearchParams& sp, cudaStream_t st) {
    auto kern = k_rowfft_stats<N, exact_stats<N>()>;
    const size_t smem = smem_pass2<N>(sp.nbins);
    { const int rc_a = ensure_smem_attr(p, (const void*)kern, smem); if (rc_a != RF_OK) return rc_a; }
    kern<<<dim3(sp.rsplit, (sp.n_img + 1) / 2), kThreads, smem, st>>>(sp);
    RF_CUDA_CHECK(cudaGetLastError());
    return RF_OK;
}

// Event bracketing for per-kernel timing: `kind` is the kernel that ran SINCE the previous
// mark (-1 = none: a start mark); 0 = grid + column FFT, 1 = row FFT + statistics, 2 = prep.
int mark(rf_plan* p, cudaStream_t st, int kind) {
    if (!p->profile) return RF_OK;
    if (p->n_events_used == (int)p->events.size()) {
        cudaEvent_t e;
        RF_CUDA_CHECK(cudaEventCreate(&e));
        p->events.push_back(e);
        p->event_kind.push_back(-1);
    }
    p->event_kind[p->n_events_used] = kind;
    RF_CUDA_CHECK(cudaEventRecord(p->events[p->n_events_used++], st));
    return RF_OK;
}

int launch_batch(rf_plan* p, const SearchParams& sp, cudaStream_t st) {
    int rc;
    if ((rc = mark(p, st, -1)) != RF_OK) return rc;
    switch (p->npix) {
#define RF_CASE(N, NCOL)                                                                    \
    case N:                                                                                 \
        if ((rc = launch_pass1_npol<N, NCOL>(p, sp, p->nchan, p->npol, st)) != RF_OK) return rc; \
        if ((rc = mark(p, st, 0)) != RF_OK) return rc;                                      \
        if ((rc = launch_pass2<N>(p, sp, st)) != RF_OK) return rc;                             \
        return mark(p, st, 1);
        RF_CASE(64, 16)
        RF_CASE(128, 16)
        RF_CASE(256, 16)
        RF_CASE(512, 16)
        RF_CASE(1024, 8)
        RF_CASE(2048, 4)
        RF_CASE(4096, 4)
#undef RF_CASE
    }
    set_error("unsupported npix %d", p->npix);
    return RF_ERR_ARG;
}

// ---------------------------------------------------------------- boxcar-tree path
// 2048 bins at every size: the quantile error of the interpolated histogram shrinks with the pixel count (B1), and at
// N >= 2048 (one 32-bit counter per bin and image) 4096 bins would cost the second row-pass CTA per SM.  Two
// bank-partitioned copies of 1024 bins over +-1.75 sigma_rms (same bin width, lanes 0-15 / 16-31 on even / odd banks) were
// measured SLOWER: row pass 19.6 vs 19.15 ms at 512^2, 728 vs 697 ms at 1024^2, 307 vs 298 ms at 4096^2.
template <int N> int tree_nbins(int) { return 2048; }

template <int N> size_t smem_tree1(int ntiles) {
    return (size_t)ntiles * (fft_padded_size(N) + 1) * sizeof(float2) + FftCfg<N>::TW_TOTAL * sizeof(float2) +
           (size_t)ntiles * FftCfg<N>::TPF * sizeof(uint32_t);
}
template <int N> constexpr int tree2_threads() { return N >= 2048 ? 256 : kThreads2; }
template <int N, int TB> size_t smem_tree2(int nbins, int cpad, int nthreads, bool zm, bool rp) {
    const size_t g2 = nthreads / FftCfg<N>::TPF;
    const size_t xb = g2 * fft_padded_size(N) * sizeof(float2);
    const size_t fin = (size_t)2 * nbins * sizeof(uint32_t);
    // staged items: one per transform group ((row, pair), or a double row with the row-pair hand-off)
    const size_t stg = rp ? g2 * (size_t)2 * cpad : g2 * (size_t)(zm ? row_stage_pitch<N, true>(cpad) : row_stage_pitch<N, false>(cpad));
    return std::max(xb, fin) + (FftCfg<N>::TW_TOTAL + kTwpSize) * sizeof(float2) + stg * sizeof(float4) +
           (size_t)(N >= 2048 ? 2 * TB - 1 : TB) * nbins * sizeof(uint32_t) + 80 * 4 + (size_t)2 * (nthreads / 32) * (2 * TB - 1) * 4;
}

// power variant of the row pass (periodicity search): 512 threads, one 32-bit histogram per pair = TB/2 images
template <int N, int TB> size_t smem_tree2_power(int nbins, int cpad) {
    const size_t g2 = kThreads2 / FftCfg<N>::TPF;
    const size_t xb = g2 * fft_padded_size(N) * sizeof(float2);
    const size_t fin = (size_t)2 * nbins * sizeof(uint32_t);
    return std::max(xb, fin) + FftCfg<N>::TW_TOTAL * sizeof(float2) + g2 * cpad * sizeof(float4) +
           (size_t)(TB / 2) * nbins * sizeof(uint32_t) + 64 * 4 + (size_t)2 * kWarps2 * TB * 4;
}

// rp: row-pair hand-off (N >= 2048 with TB = 2, see k_tree_colfft)
template <int N, int TB> constexpr bool row_pair_layout() { return N >= 2048 && TB == 2; }

template <int N, int TB, int NT2>
int launch_row_stats(rf_plan* p, const TreeParams& tp, bool zm, bool rp, cudaStream_t st) {
    void (*kern)(const TreeParams) = zm ? k_tree_rowfft_stats<N, TB, NT2, true, false> : k_tree_rowfft_stats<N, TB, NT2, false, false>;
    const int nthreads = NT2;
    if constexpr (row_pair_layout<N, TB>()) {
        if (rp) kern = zm ? k_tree_rowfft_stats<N, TB, NT2, true, true> : k_tree_rowfft_stats<N, TB, NT2, false, true>;
    }
    const size_t smem = smem_tree2<N, TB>(tp.nbins, tp.cpad, nthreads, zm, rp);
    int rc = ensure_smem_attr(p, (const void*)kern, smem);
    if (rc != RF_OK) return rc;
    kern<<<dim3(tp.n_blk), nthreads, smem, st>>>(tp);
    RF_CUDA_CHECK(cudaGetLastError());
    return RF_OK;
}

// event kinds: 0 = grid + column FFT (generic pass 1 / tree column FFT), 1 = row FFT + statistics,
// 2 = Stokes-I transpose, 3 = tree gather
template <int N, int TB, int NCOL, int QH>
int launch_tree(rf_plan* p, const TreeParams& tp, cudaStream_t st) {
    int rc;
    {
        auto kern = tp.part_major ? k_tree_gather<TB, true> : k_tree_gather<TB, false>;
        const size_t smem = (size_t)p->nchan * sizeof(int) + (size_t)kWarpsPerCta * kGatherBlocks * (2 * TB - 1) * sizeof(float);
        if (tp.n_blk % kGatherBlocks) { set_error("internal: block count %d of a tree launch is not a multiple of %d", tp.n_blk, kGatherBlocks); return RF_ERR_STATE; }
        if ((rc = mark(p, st, -1)) != RF_OK) return rc;
        const dim3 grid = tp.part_major ? dim3(tp.n_blk / kGatherBlocks, tp.n_parts) : dim3(tp.n_parts, tp.n_blk / kGatherBlocks);
        kern<<<grid, kThreads, smem, st>>>(tp);
        RF_CUDA_CHECK(cudaGetLastError());
        if ((rc = mark(p, st, 3)) != RF_OK) return rc;
    }
    // row-pair hand-off (one column per column-pass CTA, three CTAs per SM): transient search at N >= 2048 with TB = 2;
    // the periodicity search keeps the plain layout its power kernel reads
    const bool rp = row_pair_layout<N, TB>() && tp.zero_row < 0;
    bool dft = false;
    if constexpr (row_pair_layout<N, TB>()) {
        // pruned DFT over the occupied cells of every uv column (k_tree_coldft); units of N/16 threads = (column, pair),
        // a CTA keeps one column group for tune_col_dft blocks of the launch.  Only with the row-pair hand-off, where two
        // lanes fill a 32-byte sector: with the plain layout (TB = 4, or the periodicity search) every lane writes a lone
        // 16-byte piece and the kernel measured 18.7 ms against 6.75 ms for the FFTs (npix 2048, TB = 4).
        constexpr int M1 = N / 16, PAIRS = TB / 2;
        constexpr int NP = (256 / (M1 * NCOL) >= PAIRS) ? PAIRS : (256 / (M1 * NCOL) >= 1 ? 256 / (M1 * NCOL) : 1);
        static_assert(PAIRS % NP == 0, "the pairs of a block split evenly over blockIdx.z");
        const size_t smem = (size_t)kDftStages * (tp.ncmax + 1) * TB * sizeof(float2) + (size_t)tp.dft_max_blk * sizeof(int);
        // a geometry with a very full column group (the buffers of its cells must leave room for two CTAs per SM) keeps the FFTs
        dft = rp && p->tune_col_dft > 0 && tp.dft_blk != nullptr && smem <= (size_t)100 * 1024;
        if (dft) {
            void (*kern)(const TreeParams, int) = k_tree_coldft<N, TB, NCOL, NP>;
            const int spc = p->tune_col_dft;
            { const int rc_a = ensure_smem_attr(p, (const void*)kern, smem); if (rc_a != RF_OK) return rc_a; }
            kern<<<dim3(tp.ngroups, (tp.n_blk + spc - 1) / spc, PAIRS / NP), M1 * NCOL * NP, smem, st>>>(tp, spc);
            RF_CUDA_CHECK(cudaGetLastError());
            if ((rc = mark(p, st, 0)) != RF_OK) return rc;
        }
    }
    if (!dft) {
        constexpr int NTH = (N >= 4096 && QH * NCOL > 2) ? 512 : kThreads;   // 4 tiles of 4096: two concurrent transforms
        void (*kern)(const TreeParams) = k_tree_colfft<N, TB, NCOL, QH, NTH, false>;
        if constexpr (row_pair_layout<N, TB>()) { if (rp) kern = k_tree_colfft<N, TB, NCOL, QH, NTH, true>; }
        const size_t smem = smem_tree1<N>(QH * NCOL);
        { const int rc_a = ensure_smem_attr(p, (const void*)kern, smem); if (rc_a != RF_OK) return rc_a; }
        kern<<<dim3(tp.ngroups, tp.n_blk, TB / QH), NTH, smem, st>>>(tp);
        RF_CUDA_CHECK(cudaGetLastError());
        if ((rc = mark(p, st, 0)) != RF_OK) return rc;
    }
    if (tp.zero_row >= 0) {    // periodicity search: every pair is one complex image, searched in power
        auto kern = k_tree_rowfft_power<N, TB>;
        const size_t smem = smem_tree2_power<N, TB>(tp.nbins, tp.cpad);
        { const int rc_a = ensure_smem_attr(p, (const void*)kern, smem); if (rc_a != RF_OK) return rc_a; }
        kern<<<dim3(tp.n_blk), kThreads2, smem, st>>>(tp);
        RF_CUDA_CHECK(cudaGetLastError());
        return mark(p, st, 1);
    }
    {
        // half planes within 6/16 of the row (always, with the default cell: |u| <= N/3, A13) take the pruned transform
        const bool zm = tp.ncol <= 6 * FftCfg<N>::TPF;
        if ((rc = launch_row_stats<N, TB, tree2_threads<N>()>(p, tp, zm, rp, st)) != RF_OK) return rc;
        if ((rc = mark(p, st, 1)) != RF_OK) return rc;
    }
    return RF_OK;
}

int launch_tree_batch(rf_plan* p, TreeParams& tp, cudaStream_t st, int tb = 0) {
    if (tb == 0) tb = p->tree_tb;
    const int key = p->npix * 16 + tb;
    switch (key) {
#define RF_TCASE(N, TB, NCOL, QH) case N * 16 + TB: tp.nbins = tree_nbins<N>(TB); return launch_tree<N, TB, NCOL, QH>(p, tp, st);
        RF_TCASE(256, 2, 16, 2) RF_TCASE(256, 4, 8, 4) RF_TCASE(256, 8, 4, 8)
        RF_TCASE(512, 2, 8, 2) RF_TCASE(512, 4, 4, 4) RF_TCASE(512, 8, 2, 4)
        RF_TCASE(1024, 2, 4, 2) RF_TCASE(1024, 4, 2, 4) RF_TCASE(1024, 8, 2, 4)
        RF_TCASE(2048, 2, 1, 2) RF_TCASE(2048, 4, 2, 2)
        RF_TCASE(4096, 2, 1, 2) RF_TCASE(4096, 4, 2, 2)
#undef RF_TCASE
    }
    set_error("unsupported tree configuration npix %d tb %d", p->npix, tb);
    return RF_ERR_ARG;
}

// Stokes-I transpose of the integrations [t_lo, t_hi) (multiples of 32; t_hi = tpitch covers the zero pad)
int launch_prep_rows(rf_plan* p, const void* vis, cudaStream_t st, int t_lo, int t_hi) {
    const int nelem = p->nbl * p->nchan;
    const float2* mi = p->meansub ? p->ws.mean_i : nullptr;
    dim3 grid((nelem + 31) / 32, (t_hi - t_lo + 31) / 32), block(32, 8);
    const float* v = reinterpret_cast<const float*>(vis);
    int rc;
    if ((rc = mark(p, st, -1)) != RF_OK) return rc;
    switch (p->npol) {
        case 1: k_stokes_transpose<1><<<grid, block, 0, st>>>(v, p->ws.visI, mi, p->nint, nelem, p->tpitch, t_lo); break;
        case 2: k_stokes_transpose<2><<<grid, block, 0, st>>>(v, p->ws.visI, mi, p->nint, nelem, p->tpitch, t_lo); break;
        default: k_stokes_transpose<4><<<grid, block, 0, st>>>(v, p->ws.visI, mi, p->nint, nelem, p->tpitch, t_lo); break;
    }
    RF_CUDA_CHECK(cudaGetLastError());
    return mark(p, st, 2);
}
int launch_prep(rf_plan* p, const void* vis, cudaStream_t st) { return launch_prep_rows(p, vis, st, 0, p->tpitch); }

TreeParams tree_params(rf_plan* p) {
    TreeParams tp{};
    tp.visI = p->ws.visI;
    tp.delay = p->d.delay;
    tp.entries = p->d.tree.entries;
    tp.stream_iter = p->d.tree.stream_iter;
    tp.stream_cell = p->d.tree.stream_cell;
    tp.cells = p->d.tree.cells;
    tp.group_cell = p->d.tree.group_cell;
    tp.cellsum = p->ws.cellsum;
    tp.n_cells = p->d.tree.n_cells;
    tp.n_streams = p->d.tree.n_streams;
    tp.n_parts = p->d.tree.n_parts;
    tp.twiddles = p->d.twiddles;
    tp.twp = p->d.twp;
    tp.ncmax = p->d.tree.max_group_cells;
    tp.dft_max_blk = p->d.tree.dft_max_blk;
    tp.dft_blk = p->d.tree.dft_blk;
    tp.dft_off = p->d.tree.dft_off;
    tp.part_major = p->tune_gather_order;
    tp.Ht = p->ws.Ht;
    tp.sumsq = p->ws.sumsq_t;
    tp.counters = p->ws.counters;
    tp.dbg_img = -1;
    tp.dbg_slot = 0;
    tp.zero_row = -1;
    tp.dec = 1;
    tp.phase_stride = 0;
    tp.slab_stride = 0;
    tp.tpitch = p->tpitch;
    tp.nchan = p->nchan;
    tp.ncol = p->ncol;
    tp.cpad = p->d.tree.cpad;
    tp.ngroups = p->d.tree.ngroups;
    for (int l = 0; l < 4; l++) tp.dt_idx[l] = p->tree_dt_idx[l];
    tp.norm = p->n_kept > 0 ? (float)(1.0 / (2.0 * (double)p->n_kept * (double)p->npol)) : 0.f;
    tp.threshold = p->threshold;
    return tp;
}

// Widths off the tree (B7): the phase-decimated boxcar sums of width dts[k] from the Stokes-I array (once per segment) ...
int launch_phase_sum(rf_plan* p, int k, cudaStream_t st) {
    const int dt = p->dts[k], pitch = p->aux_pitch[k], nelem = p->nbl * p->nchan;
    float2* arr = p->ws.visS + p->ws.aux_off[k];
    int rc;
    if ((rc = mark(p, st, -1)) != RF_OK) return rc;
    int JC = 8;
    const size_t psm = phase_sum_smem(dt, &JC);
    if ((rc = ensure_smem_attr(p, (const void*)k_phase_sum, psm)) != RF_OK) return rc;
    k_phase_sum<<<dim3(nelem, (pitch + JC - 1) / JC), 256, psm, st>>>(p->ws.visI, arr, dt, p->tpitch, pitch, nelem, JC);
    RF_CUDA_CHECK(cudaGetLastError());
    return mark(p, st, 2);
}
// ... and the parameters with which the unchanged tree kernels search that array: level 0 of the tree = the width itself
TreeParams aux_tree_params(rf_plan* p, const TreeParams& tp, int k) {
    const int dt = p->dts[k], pitch = p->aux_pitch[k], nelem = p->nbl * p->nchan;
    TreeParams t2 = tp;
    t2.entries = p->d.aux_entries[k];
    t2.visI = p->ws.visS + p->ws.aux_off[k];
    t2.dec = dt;
    t2.phase_stride = (uint32_t)((size_t)(nelem + 1) * pitch);
    t2.dt_idx[0] = k;
    for (int l = 1; l < 4; l++) t2.dt_idx[l] = -1;
    t2.norm = tp.norm / (float)dt;
    return t2;
}

// Device buffers only ever grow (25 % headroom): the sizes follow the gridding lists, which change with every
// rf_plan_set_uvw (streaming: once per segment), and a cudaFree / cudaMalloc pair synchronises the device.
template <class T> int grow(T** ptr, size_t* cap, size_t need, bool zero = false) {
    if (*ptr && *cap >= need) return RF_OK;
    cudaFree(*ptr);
    *ptr = nullptr;
    const size_t want = need + need / 4 + 16;
    RF_CUDA_CHECK(cudaMalloc((void**)ptr, want * sizeof(T)));
    *cap = want;
    if (zero) RF_CUDA_CHECK(cudaMemset(*ptr, 0, want * sizeof(T)));
    return RF_OK;
}

int ensure_tree_workspace(rf_plan* p) {
    if (p->tree_tb == 0) return RF_OK;
    Workspace& w = p->ws;
    // one extra, all-zero series after the last (baseline, channel): the padding entries of the gather read it
    const size_t visI_elems = ((size_t)p->nbl * p->nchan + 1) * p->tpitch;
    if (!w.visI || w.visI_elems != visI_elems) {
        cudaFree(w.visI); w.visI = nullptr;
        RF_CUDA_CHECK(cudaMalloc((void**)&w.visI, visI_elems * sizeof(float2)));
        RF_CUDA_CHECK(cudaMemset(w.visI, 0, visI_elems * sizeof(float2)));
        w.visI_elems = visI_elems;
    }
    const size_t h_per_blk = (size_t)p->npix * p->d.tree.cpad * p->tree_tb;   // float2 elements
    int blk_batch = p->user_batch > 0 ? std::max(1, p->user_batch / p->tree_tb) : 0;
    if (blk_batch <= 0) {
        // pass 2 runs one CTA per block and per SM: whole waves of blocks per launch
        int dev = 0, sms = 148;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        // at least two blocks per SM per launch (N >= 2048 runs two row-pass CTAs per SM), bounded by 40 GB
        const size_t budget = std::min<size_t>((size_t)40 << 30,
                                               std::max<size_t>((size_t)4 << 30, (size_t)2 * sms * h_per_blk * sizeof(float2)));
        blk_batch = (int)std::min<size_t>(4096, std::max<size_t>(1, budget / (h_per_blk * sizeof(float2))));
        if (blk_batch > sms) blk_batch -= blk_batch % sms;
    }
    blk_batch = std::max(kGatherBlocks, blk_batch / kGatherBlocks * kGatherBlocks);          // launches hold whole gather groups
    w.blk_batch = blk_batch;
    int rc_grow = grow(&w.Ht, &w.ht_elems, h_per_blk * blk_batch);
    if (rc_grow != RF_OK) return rc_grow;
    // compact grid and Parseval partials follow the gridding lists (uvw / flags may change them)
    const size_t cs_elems = (size_t)blk_batch * std::max(1, p->d.tree.n_cells) * p->tree_tb;
    if (!w.cellsum || w.cs_elems < cs_elems) {
        cudaFree(w.cellsum); w.cellsum = nullptr;
        RF_CUDA_CHECK(cudaMalloc((void**)&w.cellsum, (cs_elems + cs_elems / 8) * sizeof(float2)));
        w.cs_elems = cs_elems + cs_elems / 8;
    }
    const size_t ss_elems = (size_t)blk_batch * (2 * p->tree_tb - 1) * std::max(1, p->d.tree.n_parts);
    if (!w.sumsq_t || w.ss_elems < ss_elems) {
        cudaFree(w.sumsq_t); w.sumsq_t = nullptr;
        RF_CUDA_CHECK(cudaMalloc((void**)&w.sumsq_t, (ss_elems + ss_elems / 8) * sizeof(float)));
        w.ss_elems = ss_elems + ss_elems / 8;
    }
    if (!w.dbg_block) RF_CUDA_CHECK(cudaMalloc((void**)&w.dbg_block, kGatherBlocks * sizeof(BlockDesc)));
    // phase-decimated sum arrays of the widths off the tree (configure_tree decided which): one after the other
    w.aux_off.assign(p->ndt + 1, 0);
    for (int k = 0; k < p->ndt; k++)
        w.aux_off[k + 1] = w.aux_off[k] + (p->aux_width[k] ? (size_t)p->dts[k] * ((size_t)p->nbl * p->nchan + 1) * p->aux_pitch[k] : 0);
    const size_t need = w.aux_off[p->ndt];
    if (need > 0 && (!w.visS || w.visS_elems < need)) {
        cudaFree(w.visS); w.visS = nullptr;
        RF_CUDA_CHECK(cudaMalloc((void**)&w.visS, need * sizeof(float2)));
        RF_CUDA_CHECK(cudaMemset(w.visS, 0, need * sizeof(float2)));      // incl. the all-zero series of every phase
        w.visS_elems = need;
    }
    return RF_OK;
}

SearchParams base_params(rf_plan* p, const void* vis) {
    SearchParams sp{};
    sp.vis = reinterpret_cast<const float*>(vis);
    sp.mean_i = p->meansub ? p->ws.mean_i : nullptr;
    sp.visI = nullptr;     // set by the caller once the Stokes-I transpose of this segment has been enqueued
    sp.tpitch = p->tpitch;
    sp.delay = p->d.delay;
    sp.entries = p->d.gen.entries;
    sp.warp_chunk = p->d.gen.warp_chunk;
    sp.twiddles = p->d.twiddles;
    sp.H = p->ws.H;
    sp.sumsq = p->ws.sumsq;
    sp.hist = p->ws.hist;
    sp.peak_val = p->ws.peak_val;
    sp.peak_pos = p->ws.peak_pos;
    sp.ticket = p->ws.ticket;
    sp.counters = p->ws.counters;
    sp.nchan = p->nchan;
    sp.ncol = p->ncol;
    sp.cpad = p->d.gen.cpad;
    sp.ngroups = p->d.gen.ngroups;
    sp.nbins = p->nbins;
    sp.rsplit = p->ws.rsplit;
    sp.row_floats = (long long)p->nbl * p->nchan * p->npol * 2;
    sp.norm = p->n_kept > 0 ? (float)(1.0 / (2.0 * (double)p->n_kept * (double)p->npol)) : 0.f;
    sp.threshold = p->threshold;
    return sp;
}

}  // namespace

void free_workspace(rf_plan* p) {
    Workspace& w = p->ws;
    cudaFree(w.H); cudaFree(w.sumsq); cudaFree(w.hist); cudaFree(w.peak_val); cudaFree(w.peak_pos);
    cudaFree(w.ticket); cudaFree(w.counters); cudaFree(w.dbg_desc);
    cudaFree(w.visI); cudaFree(w.Ht); cudaFree(w.sumsq_t); cudaFree(w.cellsum); cudaFree(w.dbg_block);
    cudaFree(w.mean_partial); cudaFree(w.mean_p); cudaFree(w.mean_i);
    cudaFree(w.visS);
    cudaFree(w.slab); cudaFree(w.pblocks); cudaFree(w.zero_delay); cudaFree(w.time_tw);
    w = Workspace{};
}

// Batch = images whose half-plane hand-off fits a fixed workspace budget; row split chosen so that
// pass 2 launches at least two CTAs per SM.  The per-image buffers exist only when the plan (or the debug hook)
// sends images down that path.
int ensure_workspace(rf_plan* p, bool need_generic) {
    Workspace& w = p->ws;
    if (!p->d.twiddles) {
        float2 tw[16 + 256];
        host_twiddles(p->npix, tw);
        RF_CUDA_CHECK(cudaMalloc((void**)&p->d.twiddles, sizeof(tw)));
        RF_CUDA_CHECK(cudaMemcpy(p->d.twiddles, tw, sizeof(tw), cudaMemcpyHostToDevice));
        float2 twp[kTwpSize];
        host_twiddle_powers(twp);
        RF_CUDA_CHECK(cudaMalloc((void**)&p->d.twp, sizeof(twp)));
        RF_CUDA_CHECK(cudaMemcpy(p->d.twp, twp, sizeof(twp), cudaMemcpyHostToDevice));
    }
    if (!w.counters) {
        RF_CUDA_CHECK(cudaMalloc((void**)&w.counters, 4 * sizeof(int32_t)));
        RF_CUDA_CHECK(cudaMemset(w.counters, 0, 4 * sizeof(int32_t)));
        RF_CUDA_CHECK(cudaMalloc((void**)&w.dbg_desc, sizeof(ImgDesc)));
    }
    if (!need_generic) return RF_OK;
    const size_t h_per_img = (size_t)p->npix * p->d.gen.cpad;    // float2 elements
    int batch = p->user_batch;
    if (batch <= 0) {
        // Measured on B200 (L-band): larger batches win (fewer launch tails) even though the
        // hand-off no longer fits L2: 237 ms at 256 images, 191 ms at 1024, 187 ms at 4096.
        const size_t budget = (size_t)3 << 30;                   // bytes of H workspace
        batch = (int)std::min<size_t>(4096, std::max<size_t>(2, budget / (h_per_img * sizeof(float2))));
    }
    batch = std::max(2, batch & ~1);
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int max_split = std::max(1, (int)((long long)p->npix * p->npix / 4096));
    int rsplit = 1;
    while ((batch / 2) * rsplit < 2 * sms && rsplit * 2 <= max_split) rsplit *= 2;
    if (p->npix <= 128) rsplit = 1;                              // exact statistics keep whole images per CTA
    p->nbins = p->npix <= 256 ? 4096 : 2048;
    w.batch = batch;
    w.rsplit = rsplit;
    int rc;
    if ((rc = grow(&w.H, &w.cap_H, h_per_img * batch)) != RF_OK) return rc;
    if ((rc = grow(&w.sumsq, &w.cap_sumsq, (size_t)batch * p->d.gen.ngroups)) != RF_OK) return rc;
    if ((rc = grow(&w.hist, &w.cap_hist, (size_t)batch * p->nbins, true)) != RF_OK) return rc;   // kernels leave it zeroed
    if ((rc = grow(&w.peak_val, &w.cap_peak_val, (size_t)batch * rsplit)) != RF_OK) return rc;
    if ((rc = grow(&w.peak_pos, &w.cap_peak_pos, (size_t)batch * rsplit)) != RF_OK) return rc;
    return grow(&w.ticket, &w.cap_ticket, (size_t)(batch / 2), true);
}

int launch_search(rf_plan* p, const void* vis, cudaStream_t st, rf_cand_out* out, const HostFeed* feed) {
    int rc = ensure_workspace(p, p->n_gen_images > 0);
    if (rc == RF_OK) rc = ensure_tree_workspace(p);
    if (rc != RF_OK) return rc;
    RF_CUDA_CHECK(cudaMemsetAsync(out->count, 0, sizeof(int32_t), st));
    RF_CUDA_CHECK(cudaMemsetAsync(p->ws.counters, 0, 4 * sizeof(int32_t), st));
    p->last_launches = 0;
    p->n_events_used = 0;
    if (p->n_kept == 0) return RF_OK;      // nothing gridded: every image is zero, snr := 0
    if (p->meansub) {                      // prep (8f-1): time means, subtracted on the fly by the readers
        if ((rc = mark(p, st, -1)) != RF_OK) return rc;
        if ((rc = launch_time_mean(p, vis, st)) != RF_OK) return rc;
        if ((rc = mark(p, st, 2)) != RF_OK) return rc;
        p->last_launches += 2;
    }
    // ---- power-of-two widths: blocks of TB integrations through the boxcar tree
    if (p->tree_tb > 0 && p->n_blocks > 0) {
        // Stokes-I transpose of the rows a launch needs, as they become available: the whole segment at once
        // for a device-resident segment, chunk by chunk behind the upload for rf_search_host (blocks are sorted
        // by the last integration they read, build_image_list)
        int rows_ready = 0;
        auto need_rows = [&](int rows) -> int {
            rows = std::min(rows, p->tpitch);
            while (rows_ready < rows) {
                int hi = p->tpitch;
                if (feed) {
                    const int c = rows_ready / feed->rows_per_chunk;
                    if (c < feed->n_chunks) RF_CUDA_CHECK(cudaStreamWaitEvent(st, feed->chunk_done[c], 0));
                    if (c + 1 < feed->n_chunks) hi = (c + 1) * feed->rows_per_chunk;
                }
                int r = launch_prep_rows(p, vis, st, rows_ready, hi);
                if (r != RF_OK) return r;
                p->last_launches += 1;
                rows_ready = hi;
            }
            return RF_OK;
        };
        TreeParams tp = tree_params(p);
        tp.cand_items = out->items;
        tp.cand_count = out->count;
        tp.cand_capacity = out->capacity;
        // behind an upload the launches start small (two waves of row-pass CTAs), so that the first ones wait for
        // few integrations; once a launch needs the whole segment anyway the batches are full-sized.  Measured at L-band
        // (end to end per segment, two runs): launches of 74 blocks 61.2 / 60.0 ms, 148 (one wave) 44.8 / 43.7, 296 44.6 / 43.1,
        // 592 46.0 / 44.4, the blocks that become searchable with each uploaded chunk 45.6.  The floor of searching behind
        // the upload is about 40 ms: half-way through the 28 ms upload only 27 % of the work is searchable (a DM trial
        // needs its whole sweep), so the GPU idles early and finishes late.  rf_plan_set_tuning(RF_TUNE_FEED_BATCH, n).
        int small = p->ws.blk_batch;
        if (feed) {
            int dev = 0, sms = 148;
            cudaGetDevice(&dev);
            cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
            small = std::min(small, 2 * sms) / kGatherBlocks * kGatherBlocks;
            if (p->tune_feed_batch > 0) small = std::max(kGatherBlocks, std::min(p->ws.blk_batch, p->tune_feed_batch) / kGatherBlocks * kGatherBlocks);
        }
        for (int64_t base = 0; base < p->n_blocks;) {
            int n = (int)std::min<int64_t>(p->ws.blk_batch, p->n_blocks - base);
            if (feed && p->h_block_deadline[base + std::min(n, small) - 1] < p->nint) n = std::min(n, small);
            tp.blocks = p->d.blocks + base;
            tp.n_blk = n;
            if ((rc = need_rows(p->h_block_deadline[base + n - 1])) != RF_OK) return rc;
            if ((rc = launch_tree_batch(p, tp, st)) != RF_OK) return rc;
            p->last_launches += 3;
            base += n;
        }
        if ((rc = need_rows(p->tpitch)) != RF_OK) return rc;      // widths off the tree read the whole array
        // ---- widths off the tree (B7): phase-decimated boxcar sums once per segment, then the same three kernels
        //      on blocks of TB consecutive OUTPUT integrations (level 0 of the tree = the width itself)
        for (int k = 0; k < p->ndt; k++) {
            const int64_t nb2 = p->aux_first[k + 1] - p->aux_first[k];
            if (!p->aux_width[k] || nb2 == 0) continue;
            if ((rc = launch_phase_sum(p, k, st)) != RF_OK) return rc;
            p->last_launches += 1;
            TreeParams t2 = aux_tree_params(p, tp, k);
            for (int64_t base = 0; base < nb2; base += p->ws.blk_batch) {
                t2.blocks = p->d.blocks2 + p->aux_first[k] + base;
                t2.n_blk = (int)std::min<int64_t>(p->ws.blk_batch, nb2 - base);
                if ((rc = launch_tree_batch(p, t2, st)) != RF_OK) return rc;
                p->last_launches += 3;
            }
        }
    }
    // ---- every other width: one gridding + transform per image
    SearchParams sp = base_params(p, vis);
    if (p->tree_tb > 0 && p->n_blocks > 0) {
        sp.visI = p->ws.visI;     // transposed above for the tree path
    }
    sp.cand_items = out->items;
    sp.cand_count = out->count;
    sp.cand_capacity = out->capacity;
    for (int64_t base = 0; base < p->n_gen_images; base += p->ws.batch) {
        sp.images = p->d.images + base;
        sp.n_img = (int)std::min<int64_t>(p->ws.batch, p->n_gen_images - base);
        if ((rc = launch_batch(p, sp, st)) != RF_OK) return rc;
        p->last_launches += 2;
    }
    return RF_OK;
}

int launch_debug_image(rf_plan* p, const void* vis, int dm_idx, int dt_idx, int t_idx,
                       float* image_dev, rf_cand* stats_dev, cudaStream_t st) {
    int rc = ensure_workspace(p, true);
    if (rc == RF_OK) rc = ensure_tree_workspace(p);
    if (rc == RF_OK && p->meansub && p->n_kept > 0) rc = launch_time_mean(p, vis, st);
    if (rc != RF_OK) return rc;
    for (int l = 0; l < 4 && p->tree_tb > 0 && p->n_kept > 0; l++) {
        if (p->tree_dt_idx[l] != dt_idx) continue;
        // the image is node (l, i) of block tb of this DM
        const int per = p->tree_tb >> l;
        int nsearch = p->nint - p->h_maxdelay[dm_idx];
        if (p->span > 0) nsearch = std::min(nsearch, p->span);
        const int tb = t_idx / per;
        BlockDesc b[kGatherBlocks];                       // the block and the others of its gather group
        for (int h = 0; h < kGatherBlocks; h++) b[h] = {dm_idx, tb / kGatherBlocks * kGatherBlocks + h, nsearch, 0};
        RF_CUDA_CHECK(cudaMemcpyAsync(p->ws.dbg_block, b, sizeof(b), cudaMemcpyHostToDevice, st));
        RF_CUDA_CHECK(cudaStreamSynchronize(st));
        if ((rc = launch_prep(p, vis, st)) != RF_OK) return rc;
        TreeParams tp = tree_params(p);
        tp.blocks = p->ws.dbg_block;
        tp.n_blk = kGatherBlocks;
        tp.dbg_slot = tb % kGatherBlocks;
        tp.image_out = image_dev;
        tp.stats_out = stats_dev;
        tp.dbg_img = tree_off(p->tree_tb, l) + t_idx % per;
        tp.cand_count = nullptr;
        return launch_tree_batch(p, tp, st);
    }
    if (p->tree_tb > 0 && p->n_kept > 0 && p->aux_width[dt_idx]) {
        // a width searched on its phase-decimated sums (B7): the same kernels as rf_search, image t_idx = level-0
        // node t_idx % TB of block t_idx / TB of this (dm, width)
        const int TB = p->tree_tb, tb = t_idx / TB;
        const int nj = p->h_num_t[(size_t)dm_idx * p->ndt + dt_idx];
        BlockDesc b[kGatherBlocks];
        for (int h = 0; h < kGatherBlocks; h++) b[h] = {dm_idx, tb / kGatherBlocks * kGatherBlocks + h, nj, 0};
        RF_CUDA_CHECK(cudaMemcpyAsync(p->ws.dbg_block, b, sizeof(b), cudaMemcpyHostToDevice, st));
        RF_CUDA_CHECK(cudaStreamSynchronize(st));
        if ((rc = launch_prep(p, vis, st)) != RF_OK) return rc;
        if ((rc = launch_phase_sum(p, dt_idx, st)) != RF_OK) return rc;
        TreeParams tp = aux_tree_params(p, tree_params(p), dt_idx);
        tp.blocks = p->ws.dbg_block;
        tp.n_blk = kGatherBlocks;
        tp.dbg_slot = tb % kGatherBlocks;
        tp.image_out = image_dev;
        tp.stats_out = stats_dev;
        tp.dbg_img = t_idx % TB;
        tp.cand_count = nullptr;
        return launch_tree_batch(p, tp, st);
    }
    ImgDesc d{dm_idx, dt_idx, t_idx, p->dts[dt_idx]};
    RF_CUDA_CHECK(cudaMemcpyAsync(p->ws.dbg_desc, &d, sizeof(d), cudaMemcpyHostToDevice, st));
    RF_CUDA_CHECK(cudaStreamSynchronize(st));   // `d` lives on this stack frame (debug hook only)
    SearchParams sp = base_params(p, vis);
    sp.images = p->ws.dbg_desc;
    sp.n_img = 1;
    sp.image_out = image_dev;
    sp.stats_out = stats_dev;
    sp.cand_count = nullptr;
    if (p->n_kept == 0) {
        if (image_dev) RF_CUDA_CHECK(cudaMemsetAsync(image_dev, 0, (size_t)p->npix * p->npix * sizeof(float), st));
        if (stats_dev) RF_CUDA_CHECK(cudaMemsetAsync(stats_dev, 0, sizeof(rf_cand), st));
        return RF_OK;
    }
    return launch_batch(p, sp, st);
}

// ---------------------------------------------------------------- periodicity search (8f-3)
// Per DM trial: time transform of the dedispersed Stokes-I series of every (baseline, channel) into a
// slab of (S[k], -i S[k]) pairs, then the gather / column-FFT kernels of the boxcar-tree path on the slab
// (zero delays: it is already dedispersed) and the power variant of the row pass.  DM trials are taken in
// chunks of n_slabs so that a chunk fills the GPU for several waves.
int periodic_nt(const rf_plan* p, int dm_idx) {
    const int n = p->nint - p->h_maxdelay[dm_idx];
    if (n < 64) return 0;
    int nt = 64;
    while (nt * 2 <= n && nt < 4096) nt *= 2;
    return nt;
}

namespace {

template <int NT>
int launch_time_fft(rf_plan* p, const int32_t* delay_dm, const float2* tw, float2* slab, cudaStream_t st) {
    constexpr int G = kThreads / FftCfg<NT>::TPF;
    auto kern = k_time_fft<NT>;
    const size_t smem = ((size_t)G * fft_padded_size(NT) + FftCfg<NT>::TW_TOTAL) * sizeof(float2);
    { const int rc_a = ensure_smem_attr(p, (const void*)kern, smem); if (rc_a != RF_OK) return rc_a; }
    const int nelem = p->nbl * p->nchan;
    kern<<<(nelem + G - 1) / G, kThreads, smem, st>>>(p->ws.visI, delay_dm, tw, slab, nelem, p->nchan, p->tpitch,
                                                       p->ws.slab_pitch);
    RF_CUDA_CHECK(cudaGetLastError());
    return RF_OK;
}

int launch_time_fft_nt(rf_plan* p, int nt, int dm_idx, int slab_idx, cudaStream_t st) {
    int lg = 0;
    while ((64 << lg) < nt) lg++;
    const float2* tw = p->ws.time_tw + (size_t)lg * (16 + 256);
    const int32_t* dd = p->d.delay + (size_t)dm_idx * p->nchan;
    float2* slab = p->ws.slab + (size_t)slab_idx * ((size_t)p->nbl * p->nchan + 1) * p->ws.slab_pitch;
    switch (nt) {
        case 64: return launch_time_fft<64>(p, dd, tw, slab, st);
        case 128: return launch_time_fft<128>(p, dd, tw, slab, st);
        case 256: return launch_time_fft<256>(p, dd, tw, slab, st);
        case 512: return launch_time_fft<512>(p, dd, tw, slab, st);
        case 1024: return launch_time_fft<1024>(p, dd, tw, slab, st);
        case 2048: return launch_time_fft<2048>(p, dd, tw, slab, st);
        case 4096: return launch_time_fft<4096>(p, dd, tw, slab, st);
    }
    set_error("unsupported time-transform length %d", nt);
    return RF_ERR_ARG;
}

int ensure_periodic_workspace(rf_plan* p, int nt_max, int n_dm_live) {
    Workspace& w = p->ws;
    // the slab has the pitch of visI: the gather entries hold element * tpitch (nt_max <= nint < tpitch)
    (void)nt_max;
    const size_t per_slab = ((size_t)p->nbl * p->nchan + 1) * p->tpitch;       // incl. the all-zero series (see visI)
    const size_t budget = (size_t)6 << 30;
    int n_slabs = (int)std::min<size_t>(8, std::max<size_t>(1, budget / (per_slab * sizeof(float2))));
    n_slabs = std::max(1, std::min(n_slabs, n_dm_live));
    if (!w.slab || w.slab_elems < per_slab * n_slabs) {
        cudaFree(w.slab); w.slab = nullptr;
        RF_CUDA_CHECK(cudaMalloc((void**)&w.slab, per_slab * n_slabs * sizeof(float2)));
        RF_CUDA_CHECK(cudaMemset(w.slab, 0, per_slab * n_slabs * sizeof(float2)));
        w.slab_elems = per_slab * n_slabs;
    }
    w.n_slabs = n_slabs;
    w.slab_pitch = p->tpitch;
    if (!w.zero_delay) {
        RF_CUDA_CHECK(cudaMalloc((void**)&w.zero_delay, (size_t)p->nchan * sizeof(int32_t)));
        RF_CUDA_CHECK(cudaMemset(w.zero_delay, 0, (size_t)p->nchan * sizeof(int32_t)));
    }
    if (!w.time_tw) {
        std::vector<float2> tw((size_t)7 * (16 + 256));
        for (int i = 0; i < 7; i++) host_twiddles(64 << i, tw.data() + (size_t)i * (16 + 256));
        RF_CUDA_CHECK(cudaMalloc((void**)&w.time_tw, tw.size() * sizeof(float2)));
        RF_CUDA_CHECK(cudaMemcpy(w.time_tw, tw.data(), tw.size() * sizeof(float2), cudaMemcpyHostToDevice));
    }
    return RF_OK;
}

}  // namespace

// dbg_dm >= 0: debug hook -- only image (dbg_dm, dbg_k), power image and statistics written out.
int launch_search_periodic(rf_plan* p, const void* vis, cudaStream_t st, rf_cand_out* out, int dbg_dm, int dbg_k,
                           float* power_dev, rf_cand* stats_dev) {
    if (p->tree_tb == 0) {
        set_error("the periodicity search runs on the boxcar-tree kernels: the plan needs npix >= 256 and "
                  "a power-of-two width <= 8 in dt_list");
        return RF_ERR_STATE;
    }
    int rc = ensure_workspace(p, false);
    if (rc == RF_OK) rc = ensure_tree_workspace(p);
    if (rc != RF_OK) return rc;
    const bool dbg = dbg_dm >= 0;
    const int TB = p->tree_tb, nimg = TB / 2;
    std::vector<int> dms;                       // DM trials with a time transform, in this call
    int nt_max = 0;
    for (int d = 0; d < p->ndm; d++) {
        if (dbg && d != dbg_dm) continue;
        const int nt = periodic_nt(p, d);
        if (nt > 0) { dms.push_back(d); nt_max = std::max(nt_max, nt); }
    }
    if (out) RF_CUDA_CHECK(cudaMemsetAsync(out->count, 0, sizeof(int32_t), st));
    RF_CUDA_CHECK(cudaMemsetAsync(p->ws.counters, 0, 4 * sizeof(int32_t), st));
    p->last_launches = 0;
    p->n_events_used = 0;
    if (dms.empty() || p->n_kept == 0) {
        if (power_dev) RF_CUDA_CHECK(cudaMemsetAsync(power_dev, 0, (size_t)p->npix * p->npix * sizeof(float), st));
        if (stats_dev) RF_CUDA_CHECK(cudaMemsetAsync(stats_dev, 0, sizeof(rf_cand), st));
        return RF_OK;
    }
    if ((rc = ensure_periodic_workspace(p, nt_max, (int)dms.size())) != RF_OK) return rc;
    Workspace& w = p->ws;
    // block list of the whole call, uploaded before the first kernel (chunk c = DM trials c*n_slabs ...)
    std::vector<BlockDesc> blocks;
    std::vector<size_t> chunk_first;
    for (size_t c0 = 0; c0 < dms.size(); c0 += w.n_slabs) {
        chunk_first.push_back(blocks.size());
        const size_t c1 = std::min(dms.size(), c0 + w.n_slabs);
        for (size_t i = c0; i < c1; i++) {
            const int nt = periodic_nt(p, dms[i]);
            for (int tb = 0; tb < nt / TB; tb++) {
                if (dbg && tb / kGatherBlocks != ((dbg_k - 1) / nimg) / kGatherBlocks) continue;      // the block's gather group
                blocks.push_back({dms[i], tb, nt, (int)(i - c0)});
            }
        }
    }
    chunk_first.push_back(blocks.size());
    // uploaded only when it differs from the list already on the device (first call, debug hook, new geometry):
    // repeated searches of a plan enqueue without synchronising
    const bool same = w.pblocks && w.h_pblocks.size() == blocks.size() &&
                      memcmp(w.h_pblocks.data(), blocks.data(), blocks.size() * sizeof(BlockDesc)) == 0;
    if (!same) {
        if (!w.pblocks || w.pblocks_cap < blocks.size()) {
            cudaFree(w.pblocks); w.pblocks = nullptr;
            RF_CUDA_CHECK(cudaMalloc((void**)&w.pblocks, blocks.size() * sizeof(BlockDesc)));
            w.pblocks_cap = blocks.size();
        }
        RF_CUDA_CHECK(cudaStreamSynchronize(st));  // an earlier search on this stream may still read the old list
        RF_CUDA_CHECK(cudaMemcpy(w.pblocks, blocks.data(), blocks.size() * sizeof(BlockDesc), cudaMemcpyHostToDevice));
        w.h_pblocks = blocks;
    }
    if (p->meansub) {
        if ((rc = launch_time_mean(p, vis, st)) != RF_OK) return rc;
        p->last_launches += 2;
    }
    if ((rc = launch_prep(p, vis, st)) != RF_OK) return rc;
    p->last_launches += 1;
    TreeParams tp = tree_params(p);
    tp.visI = w.slab;
    tp.delay = w.zero_delay;
    tp.zero_row = 0;
    tp.tpitch = w.slab_pitch;
    tp.slab_stride = ((long long)p->nbl * p->nchan + 1) * w.slab_pitch;
    tp.cand_items = out ? out->items : nullptr;
    tp.cand_count = out ? out->count : nullptr;
    tp.cand_capacity = out ? out->capacity : 0;
    if (dbg) {
        tp.image_out = power_dev;
        tp.stats_out = stats_dev;
        tp.dbg_img = (dbg_k - 1) % nimg;
        tp.dbg_slot = ((dbg_k - 1) / nimg) % kGatherBlocks;
    }
    for (size_t c = 0; c + 1 < chunk_first.size(); c++) {
        const size_t c0 = c * w.n_slabs, c1 = std::min(dms.size(), c0 + w.n_slabs);
        for (size_t i = c0; i < c1; i++) {
            if ((rc = launch_time_fft_nt(p, periodic_nt(p, dms[i]), dms[i], (int)(i - c0), st)) != RF_OK) return rc;
            p->last_launches += 1;
        }
        for (size_t base = chunk_first[c]; base < chunk_first[c + 1]; base += w.blk_batch) {
            tp.blocks = w.pblocks + base;
            tp.n_blk = (int)std::min<size_t>(w.blk_batch, chunk_first[c + 1] - base);
            if ((rc = launch_tree_batch(p, tp, st)) != RF_OK) return rc;
            p->last_launches += 3;
        }
    }
    return RF_OK;
}

}  // namespace rf
