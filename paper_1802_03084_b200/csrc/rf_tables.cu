// rf_tables.cu -- plan-time tables: (a) dispersion-delay table, (c) uv-cell table and the
// uv-column binning that lets gridding accumulate in shared memory without atomics.
//
// (a) PAPER.md:45 (footnote 1): tau = 4.15 ms DM / nu^2  -> reading A1-A4:
//     delay[dm][ch] = floor(K*dm*(1/(f*f) - 1/(fmax*fmax))/t_int + 0.5), float64, no FMA.
// (c) PAPER.md:72, 84: FFT imaging without a gridding kernel -> nearest cell (reading A8).
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>

#include "rf_internal.h"

namespace rf {

namespace {

constexpr double kDispersion = 4.148808e-3;   // s GHz^2 cm^3 / pc
constexpr double kLight = 299792458.0;        // m / s

// Every operation is an explicitly rounded IEEE float64 op (no contraction to FMA), in the
// order the definition is written, so the table is bit-exact against any IEEE evaluation.
__global__ void k_delay_table(const double* __restrict__ freqs_hz, const double* __restrict__ dms,
                              int nchan, int ndm, double fmax_ghz, double inttime,
                              int32_t* __restrict__ delay) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nchan * ndm) return;
    int ch = i % nchan, d = i / nchan;
    double f = __ddiv_rn(freqs_hz[ch], 1e9);
    double a = __ddiv_rn(1.0, __dmul_rn(f, f));
    double b = __ddiv_rn(1.0, __dmul_rn(fmax_ghz, fmax_ghz));
    double x = __ddiv_rn(__dmul_rn(__dmul_rn(kDispersion, dms[d]), __dsub_rn(a, b)), inttime);
    delay[i] = (int32_t)floor(__dadd_rn(x, 0.5));
}

__global__ void k_cell_table(const double* __restrict__ uvw, const double* __restrict__ freqs_hz,
                             const float* __restrict__ weights, int nbl, int nchan, int npix,
                             double du, int32_t* __restrict__ cell, uint8_t* __restrict__ keep) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nbl * nchan) return;
    int ch = i % nchan, bl = i / nchan;
    double f = freqs_hz[ch];
    double ul = __ddiv_rn(__dmul_rn(uvw[3 * bl + 0], f), kLight);
    double vl = __ddiv_rn(__dmul_rn(uvw[3 * bl + 1], f), kLight);
    // clamp before the int conversion so absurd geometry cannot overflow int32
    double a = fmin(fmax(floor(__dadd_rn(__ddiv_rn(ul, du), 0.5)), -1.0e9), 1.0e9);
    double e = fmin(fmax(floor(__dadd_rn(__ddiv_rn(vl, du), 0.5)), -1.0e9), 1.0e9);
    int iu = (int)a, iv = (int)e;
    int half = npix / 2;
    bool ok = iu >= -half && iu < half && iv >= -half && iv < half && weights[ch] != 0.0f;
    cell[2 * i + 0] = iu;
    cell[2 * i + 1] = iv;
    keep[i] = ok ? 1 : 0;
}

// Device buffers are kept between rebuilds (capacity per pointer variable) and all plan-time
// work runs on the plan's own non-blocking stream, so rf_plan_set_uvw neither frees memory nor
// touches the legacy default stream: a rebuild does not synchronise with searches of OTHER plans
// that are in flight (streaming, config 5: two plans used alternately).
template <class T> int reserve(rf_plan* p, T** dst, size_t n) {
    size_t& cap = p->dev_cap[(void*)dst];
    const size_t bytes = n * sizeof(T);
    if (*dst && bytes <= cap) return RF_OK;
    if (*dst) { cudaFree(*dst); *dst = nullptr; cap = 0; }
    if (n == 0) return RF_OK;
    const size_t want = bytes + bytes / 4 + 256;
    if (cudaMalloc((void**)dst, want) != cudaSuccess) {
        cudaGetLastError();
        set_error("device allocation of %zu bytes failed", want);
        return RF_ERR_NOMEM;
    }
    cap = want;
    return RF_OK;
}
template <class T> int upload(rf_plan* p, T** dst, const T* src, size_t n) {
    int rc = reserve(p, dst, n);
    if (rc != RF_OK || n == 0) return rc;
    // pageable source: returns once the data is staged, so `src` may be freed by the caller
    RF_CUDA_CHECK(cudaMemcpyAsync(*dst, src, n * sizeof(T), cudaMemcpyHostToDevice, p->tab_stream));
    return RF_OK;
}

}  // namespace

int build_delay_table(rf_plan* p) {
    int rc;
    if ((rc = upload(p, &p->d.freqs, p->freqs.data(), p->freqs.size())) != RF_OK) return rc;
    if ((rc = upload(p, &p->d.dms, p->dms.data(), p->dms.size())) != RF_OK) return rc;
    size_t n = (size_t)p->ndm * p->nchan;
    if ((rc = reserve(p, &p->d.delay, n)) != RF_OK) return rc;
    double fmax = *std::max_element(p->freqs.begin(), p->freqs.end()) / 1e9;
    k_delay_table<<<(unsigned)((n + 255) / 256), 256, 0, p->tab_stream>>>(p->d.freqs, p->d.dms, p->nchan, p->ndm, fmax,
                                                        p->inttime, p->d.delay);
    RF_CUDA_CHECK(cudaGetLastError());
    p->h_delay.resize(n);
    RF_CUDA_CHECK(cudaMemcpyAsync(p->h_delay.data(), p->d.delay, n * sizeof(int32_t), cudaMemcpyDeviceToHost, p->tab_stream));
    RF_CUDA_CHECK(cudaStreamSynchronize(p->tab_stream));
    p->h_maxdelay.assign(p->ndm, 0);
    for (int d = 0; d < p->ndm; d++)
        for (int c = 0; c < p->nchan; c++)
            p->h_maxdelay[d] = std::max(p->h_maxdelay[d], p->h_delay[(size_t)d * p->nchan + c]);
    return RF_OK;
}

int build_cell_table(rf_plan* p) {
    int rc;
    if ((rc = upload(p, &p->d.uvw, p->uvw.data(), p->uvw.size())) != RF_OK) return rc;
    if ((rc = upload(p, &p->d.weights, p->weights.data(), p->weights.size())) != RF_OK) return rc;
    size_t n = (size_t)p->nbl * p->nchan;
    if ((rc = reserve(p, &p->d.cell, 2 * n)) != RF_OK) return rc;
    if ((rc = reserve(p, &p->d.keep, n)) != RF_OK) return rc;
    double du = 1.0 / (p->npix * p->cell);
    k_cell_table<<<(unsigned)((n + 255) / 256), 256, 0, p->tab_stream>>>(p->d.uvw, p->d.freqs, p->d.weights, p->nbl, p->nchan,
                                                       p->npix, du, p->d.cell, p->d.keep);
    RF_CUDA_CHECK(cudaGetLastError());
    p->h_cell.resize(2 * n);
    p->h_keep.resize(n);
    RF_CUDA_CHECK(cudaMemcpyAsync(p->h_cell.data(), p->d.cell, 2 * n * sizeof(int32_t), cudaMemcpyDeviceToHost, p->tab_stream));
    RF_CUDA_CHECK(cudaMemcpyAsync(p->h_keep.data(), p->d.keep, n, cudaMemcpyDeviceToHost, p->tab_stream));
    RF_CUDA_CHECK(cudaStreamSynchronize(p->tab_stream));
    p->n_kept = 0;
    for (size_t i = 0; i < n; i++) p->n_kept += p->h_keep[i];
    p->n_dropped = (int)n - p->n_kept;
    return RF_OK;
}

// Route every kept sample to the half plane 0 <= column <= N/2 (the other half is its
// Hermitian mirror and is never stored), sort by (column group, column, row, bl, ch), cut
// each group into kWarpsPerCta ranges at cell boundaries and pad each range to whole
// 32-lane chunks.  Inside a chunk equal cells are contiguous, so a segmented warp scan
// followed by ONE plain read-modify-write per cell replaces shared-memory atomics, and the
// summation order is fixed (bitwise reproducible grids).
int build_grid_lists(rf_plan* p) {
    const int N = p->npix, half = N / 2;
    struct Raw { uint32_t col, row, elem, ch, conj; };
    std::vector<Raw> raw;
    raw.reserve((size_t)p->n_kept + 1024);
    int maxcol = -1;
    for (int bl = 0; bl < p->nbl; bl++)
        for (int ch = 0; ch < p->nchan; ch++) {
            size_t i = (size_t)bl * p->nchan + ch;
            if (!p->h_keep[i]) continue;
            int iu = p->h_cell[2 * i], iv = p->h_cell[2 * i + 1];
            int c0 = ((iu % N) + N) % N, r0 = ((iv % N) + N) % N;
            int c1 = ((-iu % N) + N) % N, r1 = ((-iv % N) + N) % N;
            if (c0 <= half) { raw.push_back({(uint32_t)c0, (uint32_t)r0, (uint32_t)i, (uint32_t)ch, 0u}); maxcol = std::max(maxcol, c0); }
            if (c1 <= half) { raw.push_back({(uint32_t)c1, (uint32_t)r1, (uint32_t)i, (uint32_t)ch, 1u}); maxcol = std::max(maxcol, c1); }
        }
    std::sort(raw.begin(), raw.end(), [](const Raw& a, const Raw& b) {
        if (a.col != b.col) return a.col < b.col;
        if (a.row != b.row) return a.row < b.row;
        if (a.elem != b.elem) return a.elem < b.elem;
        return a.conj < b.conj;
    });
    p->ncol = std::max(1, maxcol + 1);
    p->n_entries = (int64_t)raw.size();

    auto emit = [&](GridLists& gl, int kColsPerGroup) -> int {
        gl.colgrp = kColsPerGroup;
        gl.cpad = (p->ncol + kColsPerGroup - 1) / kColsPerGroup * kColsPerGroup;
        gl.ngroups = gl.cpad / kColsPerGroup;
        std::vector<GridEntry> entries;
        std::vector<int32_t> warp_chunk(gl.ngroups * kWarpsPerCta + 1, 0);
        entries.reserve(raw.size() + (size_t)gl.ngroups * kWarpsPerCta * 32);
        size_t pos = 0;
        for (int g = 0; g < gl.ngroups; g++) {
            size_t gbeg = pos;
            while (pos < raw.size() && (int)(raw[pos].col / kColsPerGroup) == g) pos++;
            size_t gend = pos, cnt = gend - gbeg;
            size_t cut = gbeg;
            for (int w = 0; w < kWarpsPerCta; w++) {
                warp_chunk[g * kWarpsPerCta + w] = (int32_t)(entries.size() / 32);
                // ideal end of this warp's range, moved forward to the next cell boundary
                size_t want = gbeg + cnt * (w + 1) / kWarpsPerCta;
                size_t end = std::max(want, cut);
                if (w == kWarpsPerCta - 1) end = gend;
                while (end < gend && end > gbeg && raw[end].col == raw[end - 1].col && raw[end].row == raw[end - 1].row) end++;
                for (size_t s = cut; s < end; s += 32) {
                    size_t e = std::min(end, s + 32);
                    for (size_t k = s; k < s + 32; k++) {
                        GridEntry ge{0u, 0u};
                        if (k < e) {
                            const Raw& r = raw[k];
                            size_t h = k;   // first lane of this cell inside the chunk
                            while (h > s && raw[h - 1].col == r.col && raw[h - 1].row == r.row) h--;
                            bool tail = (k + 1 == e) || raw[k + 1].col != r.col || raw[k + 1].row != r.row;
                            ge.w0 = r.elem | ((uint32_t)(k - h) << 24) | (tail ? (1u << 29) : 0u) |
                                    (r.conj << 30) | (1u << 31);
                            ge.w1 = r.ch | (r.row << 12) | ((r.col % kColsPerGroup) << 24);
                        }
                        entries.push_back(ge);
                    }
                }
                cut = end;
            }
        }
        warp_chunk[gl.ngroups * kWarpsPerCta] = (int32_t)(entries.size() / 32);
        gl.n_chunks = (int64_t)entries.size() / 32;
        int rc;
        if ((rc = upload(p, &gl.entries, entries.data(), entries.size())) != RF_OK) return rc;
        return upload(p, &gl.warp_chunk, warp_chunk.data(), warp_chunk.size());
    };
    // Tree path ("time in lanes"): a warp reads LG = 32/TB entries per iteration, lane = (entry j,
    // integration q), so the TB consecutive samples of an entry are one coalesced 8*TB-byte read.
    // Cells are numbered in (column, row) order.  The gather kernel walks them in WARP STREAMS:
    // runs of consecutive cells of about kStreamIters iterations, cut at cell boundaries and padded
    // to a multiple of kTreeUnroll iterations with weight-0 entries.  A cell of n entries fills
    // ceil(n/LG) consecutive iterations of its stream; the lane accumulates over them in a register,
    // the iteration flagged END sums the LG lane groups and writes the cell sum to the compact grid
    // cellsum[block][cell][q] -- one owner per cell, fixed summation order, no atomics.  The column-FFT
    // kernel of column group g then scatters cells group_cell[g] .. group_cell[g+1] into its tiles.
    auto emit_tree = [&](TreeLists& tl, int kColsPerGroup, int LG) -> int {
        tl.colgrp = kColsPerGroup;
        tl.lg = LG;
        tl.cpad = (p->ncol + kColsPerGroup - 1) / kColsPerGroup * kColsPerGroup;
        tl.ngroups = tl.cpad / kColsPerGroup;
        std::vector<uint2> entries;
        std::vector<uint32_t> cells;
        std::vector<int32_t> stream_iter, stream_cell, group_cell(tl.ngroups + 1, 0);
        entries.reserve(raw.size() * 5 / 4 + 1024);
        int64_t iters = 0, stream_start = 0;
        // entry = (row offset of the (baseline, channel) series in visI, channel | flags)
        auto make_entry = [&](const Raw& r, uint32_t flags) { return make_uint2(r.elem * (uint32_t)p->tpitch, r.ch | flags); };
        // padding reads the all-zero series that follows the last (baseline, channel) in visI
        auto pad_entry = [&]() -> uint2 { return make_uint2((uint32_t)p->nbl * (uint32_t)p->nchan * (uint32_t)p->tpitch, 0u); };
        auto close_stream = [&]() {
            for (; (iters - stream_start) % kTreeUnroll; iters++)
                for (int j = 0; j < LG; j++) entries.push_back(pad_entry());
            stream_start = iters;
        };
        stream_iter.push_back(0);
        stream_cell.push_back(0);
        int next_group = 0;
        for (size_t c0 = 0; c0 < raw.size();) {
            size_t c1 = c0;
            while (c1 < raw.size() && raw[c1].col == raw[c0].col && raw[c1].row == raw[c0].row) c1++;
            const int n = (int)(c1 - c0), cit = (n + LG - 1) / LG;
            const int g = (int)(raw[c0].col / kColsPerGroup);
            while (next_group <= g) group_cell[next_group++] = (int32_t)cells.size();
            if (iters - stream_start > 0 && iters - stream_start + cit > kStreamIters) {
                close_stream();
                stream_iter.push_back((int32_t)iters);
                stream_cell.push_back((int32_t)cells.size());
            }
            const bool edge = raw[c0].col == 0 || (int)raw[c0].col == N / 2;
            cells.push_back(raw[c0].row | ((raw[c0].col % kColsPerGroup) << 12) | (edge ? (1u << 16) : 0u));
            for (int it = 0; it < cit; it++)
                for (int j = 0; j < LG; j++) {
                    const int k = it * LG + j;
                    const bool valid = k < n;
                    const uint32_t flags = (edge ? (1u << 28) : 0u) | (it == cit - 1 ? (1u << 29) : 0u);
                    if (valid) entries.push_back(make_entry(raw[c0 + k], flags | (raw[c0 + k].conj << 31)));
                    else { uint2 e = pad_entry(); e.y |= flags; entries.push_back(e); }
                }
            iters += cit;
            c0 = c1;
        }
        while (next_group <= tl.ngroups) group_cell[next_group++] = (int32_t)cells.size();
        close_stream();
        stream_iter.push_back((int32_t)iters);
        stream_cell.push_back((int32_t)cells.size());
        tl.n_iters = iters;
        tl.n_cells = (int)cells.size();
        tl.max_group_cells = 0;
        for (int g = 0; g < tl.ngroups; g++) tl.max_group_cells = std::max(tl.max_group_cells, group_cell[g + 1] - group_cell[g]);
        tl.n_streams = (int)stream_iter.size() - 1;
        tl.n_parts = (tl.n_streams + kWarpsPerCta - 1) / kWarpsPerCta;
        // A cell cannot be split, so streams differ in length (a 848-sample cell alone is 424 iterations at S-band) and a
        // gather CTA waits at its final barrier for its longest stream.  Streams are therefore handed out sorted by
        // length: the 8 streams of a CTA are about equally long, and the long CTAs come first in the grid.
        {
            std::vector<int> order(tl.n_streams);
            for (int i = 0; i < tl.n_streams; i++) order[i] = i;
            std::stable_sort(order.begin(), order.end(), [&](int a, int b) {
                return stream_iter[a + 1] - stream_iter[a] > stream_iter[b + 1] - stream_iter[b];
            });
            std::vector<int32_t> it2(2 * (size_t)tl.n_streams), c2(tl.n_streams);
            for (int i = 0; i < tl.n_streams; i++) {
                it2[2 * i] = stream_iter[order[i]];
                it2[2 * i + 1] = stream_iter[order[i] + 1];
                c2[i] = stream_cell[order[i]];
            }
            stream_iter.swap(it2);
            stream_cell.swap(c2);
        }
        int rc;
        // widths searched on phase-decimated sums: the same entries with that array's row pitch
        if ((int)p->d.aux_entries.size() != p->ndt) p->d.aux_entries.assign(p->ndt, nullptr);
        for (int k = 0; k < p->ndt; k++) {
            if (!p->aux_width[k]) continue;
            std::vector<uint2> e2(entries);
            for (uint2& e : e2) e.x = (e.x / (uint32_t)p->tpitch) * (uint32_t)p->aux_pitch[k];
            if ((rc = upload(p, &p->d.aux_entries[k], e2.data(), e2.size())) != RF_OK) return rc;
        }
        // List blocks of the pruned column transform (k_tree_coldft, npix >= 2048 with TB = 2), one per column group:
        //   [first entry of (column, class) k = 0 .. 16 colgrp | pad to 4 ints][entries | 4 entries of read-ahead | pad to 4]
        // entry = (row / 16) | (cell of the group + 1) << 8, sorted by (column, class = row mod 16) like the cells themselves;
        // every class is padded to an even number of entries with 0 (= the zero cell in front of the staged values).
        tl.dft_max_blk = 0;
        if (N >= 2048 && p->tree_tb == 2) {
            const int NK = kColsPerGroup * 16, hdr = (NK + 1 + 3) & ~3;
            std::vector<int32_t> blk, off(tl.ngroups + 1, 0);
            std::vector<int> cnt(NK), start(NK + 1);
            for (int g = 0; g < tl.ngroups; g++) {
                off[g] = (int32_t)blk.size();
                const int cb = group_cell[g], nc = group_cell[g + 1] - cb;
                std::fill(cnt.begin(), cnt.end(), 0);
                auto key_of = [](uint32_t m) { return (int)((m >> 12) & 0xfu) * 16 + (int)(m & 0xfu); };
                for (int i = 0; i < nc; i++) cnt[key_of(cells[cb + i])]++;
                start[0] = 0;
                for (int k = 0; k < NK; k++) start[k + 1] = start[k] + cnt[k] + (cnt[k] & 1);
                const int total = start[NK];
                const size_t base = blk.size();
                blk.resize(base + hdr + (((size_t)total + 4 + 3) & ~(size_t)3), 0);
                for (int k = 0; k <= NK; k++) blk[base + k] = start[k];
                std::fill(cnt.begin(), cnt.end(), 0);
                for (int i = 0; i < nc; i++) {
                    const uint32_t m = cells[cb + i];
                    const int k = key_of(m);
                    blk[base + hdr + start[k] + cnt[k]++] = (int32_t)(((m & 0xfffu) >> 4) | ((uint32_t)(i + 1) << 8));
                }
                tl.dft_max_blk = std::max(tl.dft_max_blk, (int)(blk.size() - base));
            }
            off[tl.ngroups] = (int32_t)blk.size();
            if ((rc = upload(p, &tl.dft_blk, blk.data(), blk.size())) != RF_OK) return rc;
            if ((rc = upload(p, &tl.dft_off, off.data(), off.size())) != RF_OK) return rc;
        }
        if ((rc = upload(p, &tl.entries, entries.data(), entries.size())) != RF_OK) return rc;
        if ((rc = upload(p, &tl.cells, cells.data(), cells.size())) != RF_OK) return rc;
        if ((rc = upload(p, &tl.stream_iter, stream_iter.data(), stream_iter.size())) != RF_OK) return rc;
        if ((rc = upload(p, &tl.stream_cell, stream_cell.data(), stream_cell.size())) != RF_OK) return rc;
        return upload(p, &tl.group_cell, group_cell.data(), group_cell.size());
    };
    int rc = emit(p->d.gen, cols_per_group(N));
    if (rc == RF_OK && p->tree_tb > 0) {
        // the pruned column transform (k_tree_coldft) walks the cells of a column class by class (row mod 16)
        std::sort(raw.begin(), raw.end(), [](const Raw& a, const Raw& b) {
            if (a.col != b.col) return a.col < b.col;
            if ((a.row & 15u) != (b.row & 15u)) return (a.row & 15u) < (b.row & 15u);
            if (a.row != b.row) return a.row < b.row;
            if (a.elem != b.elem) return a.elem < b.elem;
            return a.conj < b.conj;
        });
    }
    if (rc == RF_OK && p->tree_tb > 0) rc = emit_tree(p->d.tree, tree_cols_per_group(N, p->tree_tb), 32 / (kGatherBlocks * p->tree_tb));   // kGatherBlocks TB lanes per entry
    if (rc == RF_OK) RF_CUDA_CHECK(cudaStreamSynchronize(p->tab_stream));
    return rc;
}

// Columns per pass-1 CTA of the tree path: TB x NCOL column tiles of N points must fit ~70 KB
// of shared memory (139 KB for 4096 x 2).
int tree_cols_per_group(int npix, int tb) {
    if (npix <= 512) return (16 * 512) / (npix * tb);     // TB x NCOL = 16 tiles of 512 (32 of 256): 70 KB
    if (npix == 1024) return tb == 2 ? 4 : 2;             // 8 tiles of 1024; TB > 4 is split over blockIdx.z
    return tb == 2 ? 1 : 2;                               // TB = 2: one column x 2 integrations (row-pair hand-off, 74 KB at 4096,
                                                          // three CTAs per SM); TB = 4: 4 tiles of 2048 (70 KB) / 4096 (139 KB)
}

// Row pitch of the phase-decimated sum array of width dt: output integrations j' = t / dt of one series and phase,
// plus the read-ahead of the last block pair and of the largest delay.
int aux_pitch_of(const rf_plan* p, int dt) { return (((p->tpitch + dt - 1) / dt + kGatherBlocks * p->tree_tb + 8) + 7) & ~7; }

// Which widths off the tree are searched by the tree kernels on phase-decimated sums (B7): every width > 1 while the
// sum arrays fit kSlidingSumBudget (each is about the size of the Stokes-I array); the rest takes the per-image path.
// Dynamic shared memory of k_phase_sum for a width: in [JC*dt + dt] | sums [JC*dt padded by 1/32] float2.
size_t phase_sum_smem(int dt, int* jc_out) {
    const int JC = std::max(8, 2048 / dt);
    if (jc_out) *jc_out = JC;
    return ((size_t)JC * dt + dt + (size_t)JC * dt + (size_t)JC * dt / 32 + 2) * sizeof(float2);
}

static void decide_aux_widths(rf_plan* p) {
    p->aux_width.assign(p->ndt, 0);
    p->aux_pitch.assign(p->ndt, 0);
    if (p->tree_tb == 0 || !p->tune_aux) return;
    size_t bytes = 0;
    for (int k = 0; k < p->ndt; k++) {
        bool in_tree = false;
        for (int l = 0; l < 4; l++) in_tree |= (p->tree_dt_idx[l] == k);
        const int dt = p->dts[k];
        if (in_tree || dt <= 1 || dt >= p->nint) continue;
        const size_t need = (size_t)dt * ((size_t)p->nbl * p->nchan + 1) * aux_pitch_of(p, dt) * sizeof(float2);
        if (bytes + need > kSlidingSumBudget || need / sizeof(float2) >= (1ull << 32)) continue;
        if (phase_sum_smem(dt, nullptr) > kMaxDynSmem) continue;     // very wide boxcars: per-image path
        bytes += need;
        p->aux_width[k] = 1;
        p->aux_pitch[k] = aux_pitch_of(p, dt);
    }
}

// Loop + segment semantics (readings A6, A16): all j with
// (j+1)*dt <= min(nint - maxdelay(dm), span).
void configure_tree(rf_plan* p) {
    // which dt values ride the image-domain boxcar tree (B3)
    p->tree_tb = 0;
    for (int l = 0; l < 4; l++) p->tree_dt_idx[l] = -1;
    // every size from 256 up rides the tree (N >= 2048: 256-thread row-pass CTAs, see launch_tree);
    // rf_plan_set_tuning(RF_TUNE_TREE_MAXPIX) lowers the limit
    if (p->use_tree && p->npix >= 256 && p->npix <= p->tune_tree_maxpix) {
        // N >= 2048: the row pass keeps one 32-bit histogram per image, so TB stops at 4 there (launch_tree_batch);
        // a width of 8 then rides the phase-decimated sums (B7) like any other width off the tree
        const int tb_max = p->npix >= 2048 ? 4 : 8;
        for (int k = 0; k < p->ndt; k++) {
            const int dt = p->dts[k];
            for (int l = 0; l < 4; l++)
                if (dt == (1 << l) && dt <= tb_max && p->tree_dt_idx[l] < 0) {
                    p->tree_dt_idx[l] = k;
                    p->tree_tb = std::max(p->tree_tb, dt);
                }
        }
        if (p->tree_tb == 1) p->tree_tb = 2;      // the pair transform needs two integrations
    }
    // read-ahead of the last block group of a DM (the gather reads kGatherBlocks TB integrations per entry)
    p->tpitch = p->tree_tb ? ((p->nint + kGatherBlocks * p->tree_tb + 15) / 16) * 16 : 0;
    // gather entries hold (baseline * nchan + channel) * tpitch in 32 bits
    if (((unsigned long long)p->nbl * p->nchan + 1) * p->tpitch >= (1ull << 32)) {
        p->tree_tb = 0; p->tpitch = 0;
        for (int l = 0; l < 4; l++) p->tree_dt_idx[l] = -1;
    }
    decide_aux_widths(p);
}

int build_image_list(rf_plan* p) {
    std::vector<ImgDesc> imgs;
    std::vector<BlockDesc> blocks;
    p->h_num_t.assign((size_t)p->ndm * p->ndt, 0);
    p->vis_gridded = 0;
    p->n_images = 0;
    std::vector<int> nsearch_of(p->ndm, 0);
    std::vector<char> in_tree_dm(p->ndm, 0);
    for (int d = 0; d < p->ndm; d++) {
        int nsearch = p->nint - p->h_maxdelay[d];
        if (p->span > 0) nsearch = std::min(nsearch, p->span);
        nsearch_of[d] = nsearch;
        for (int k = 0; k < p->ndt; k++) {
            int dt = p->dts[k];
            int nj = nsearch > 0 ? nsearch / dt : 0;
            p->h_num_t[(size_t)d * p->ndt + k] = nj;
            p->n_images += nj;
            p->vis_gridded += (int64_t)nj * dt * p->n_kept;
            bool in_tree = false;
            for (int l = 0; l < 4; l++) in_tree |= (p->tree_dt_idx[l] == k);
            if (in_tree) { in_tree_dm[d] |= nj > 0; continue; }
        }
    }
    // DM trials sorted by their sweep and taken in groups of kDmGroup neighbours (both paths)
    std::vector<int> order(p->ndm);
    for (int d = 0; d < p->ndm; d++) order[d] = d;
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return p->h_maxdelay[a] < p->h_maxdelay[b]; });
    const int dm_group = std::max(1, p->tune_dm_group);
    // Image order of the per-image path: per width, DM groups, output integration j in the OUTER loop and
    // the DM trials of the group inside.  Concurrent CTAs of one column group (blockIdx.x = image) then read
    // the same (baseline, channel) rows at times a few integrations apart: the 32-byte sectors of the
    // gather are shared in L2 instead of being fetched from HBM once per image at random addresses.
    // Widths off the tree that configure_tree marked (aux_width): blocks of TB consecutive OUTPUT integrations of one
    // DM, searched by the tree kernels on the phase-decimated sum array of the width (B7); only level 0 is valid.
    p->aux_first.assign(p->ndt + 1, 0);
    std::vector<BlockDesc> blocks2;
    for (int k = 0; k < p->ndt; k++) {
        p->aux_first[k] = (int64_t)blocks2.size();
        if (!p->aux_width[k]) continue;
        for (int g0 = 0; g0 < p->ndm; g0 += dm_group) {
            const int g1 = std::min(p->ndm, g0 + dm_group);
            int max_blk = 0;
            std::vector<int> nblk(g1 - g0, 0);
            const int TB = p->tree_tb, GB = kGatherBlocks;
            for (int i = g0; i < g1; i++) {
                const int nj = p->h_num_t[(size_t)order[i] * p->ndt + k];
                nblk[i - g0] = nj > 0 ? (((nj + TB - 1) / TB) + GB - 1) / GB * GB : 0;    // blocks of TB images, whole gather groups
                max_blk = std::max(max_blk, nblk[i - g0]);
            }
            for (int tb = 0; tb < max_blk; tb += GB)
                for (int i = g0; i < g1; i++)
                    if (tb < nblk[i - g0])
                        for (int h = 0; h < GB; h++)     // nsearch field = number of valid images of this (dm, width)
                            blocks2.push_back({order[i], tb + h, p->h_num_t[(size_t)order[i] * p->ndt + k], 0});
        }
    }
    p->aux_first[p->ndt] = (int64_t)blocks2.size();
    for (int k = 0; k < p->ndt; k++) {
        bool in_tree = false;
        for (int l = 0; l < 4; l++) in_tree |= (p->tree_dt_idx[l] == k);
        if (in_tree || p->aux_width[k]) continue;
        const int dt = p->dts[k];
        for (int g0 = 0; g0 < p->ndm; g0 += dm_group) {
            const int g1 = std::min(p->ndm, g0 + dm_group);
            int max_nj = 0;
            for (int i = g0; i < g1; i++) max_nj = std::max(max_nj, p->h_num_t[(size_t)order[i] * p->ndt + k]);
            for (int j = 0; j < max_nj; j++)
                for (int i = g0; i < g1; i++)
                    if (j < p->h_num_t[(size_t)order[i] * p->ndt + k]) imgs.push_back({order[i], k, j, dt});
        }
    }
    // Block order of the tree path: DM trials sorted by their sweep and taken in groups of
    // kDmGroup neighbours; inside a group time runs in the OUTER loop.  Consecutive blocks then
    // read nearly the same window of every (baseline, channel) row (neighbouring DMs differ by a
    // few integrations of delay), so the gather is served from L2 instead of re-reading the whole
    // Stokes-I array from HBM once per DM trial.
    // Units of one DM group x one time block are then sorted by the last integration they read ("deadline"
    // = tb*TB + TB + largest sweep of the group): the search consumes the segment front to back, so
    // rf_search_host can start it while the upload of the later integrations is still in flight, and a
    // launch never needs rows beyond the deadline of its last block (h_block_deadline).
    p->h_block_deadline.clear();
    if (p->tree_tb > 0) {
        const int TB = p->tree_tb, GB = kGatherBlocks;
        // blocks per DM, rounded up to whole gather groups: the gather kernel serves GB consecutive time blocks
        // (slots GB y ... GB y + GB - 1 of a launch); padding blocks lie past the searched range, hold no valid image
        // and are skipped by the row pass
        std::vector<int> nblk(p->ndm, 0);
        for (int d = 0; d < p->ndm; d++)
            if (in_tree_dm[d]) nblk[d] = (((nsearch_of[d] + TB - 1) / TB) + GB - 1) / GB * GB;
        struct Unit { int g0, tb, deadline; };
        std::vector<Unit> units;
        for (int g0 = 0; g0 < p->ndm; g0 += dm_group) {
            const int g1 = std::min(p->ndm, g0 + dm_group);
            int max_blk = 0, sweep = 0;
            for (int i = g0; i < g1; i++)
                if (in_tree_dm[order[i]]) {
                    max_blk = std::max(max_blk, nblk[order[i]]);
                    sweep = std::max(sweep, p->h_maxdelay[order[i]]);
                }
            // a unit = kUnitBlocks consecutive time blocks of the group: neighbouring blocks share 128-byte lines
            for (int tb = 0; tb < max_blk; tb += kUnitBlocks)
                units.push_back({g0, tb, std::min(p->tpitch, (tb + kUnitBlocks) * TB + sweep)});
        }
        std::stable_sort(units.begin(), units.end(), [](const Unit& a, const Unit& b) { return a.deadline < b.deadline; });
        for (const Unit& u : units) {
            const int g1 = std::min(p->ndm, u.g0 + dm_group);
            for (int tb = u.tb; tb < u.tb + kUnitBlocks; tb += GB)
                for (int i = u.g0; i < g1; i++) {
                    const int d = order[i];
                    if (tb >= nblk[d]) continue;
                    for (int h = 0; h < GB; h++) {
                        blocks.push_back({d, tb + h, nsearch_of[d], 0});
                        p->h_block_deadline.push_back(u.deadline);
                    }
                }
        }
    }
    p->n_gen_images = (int64_t)imgs.size();
    p->n_blocks = (int64_t)blocks.size();
    // transforms actually run per search (bench.py: FFT rate under the 5 N log2 N convention): the tree kernels
    // transform every padded column of every integration of every block and run TB/2 pair transforms per row
    {
        const int64_t nb = (int64_t)blocks.size() + (int64_t)blocks2.size();
        p->n_col_fft = nb * p->tree_tb * p->d.tree.cpad + (int64_t)imgs.size() * p->d.gen.cpad;
        p->n_row_fft = nb * (p->tree_tb / 2) * p->npix + ((int64_t)imgs.size() + 1) / 2 * p->npix;
    }
    int rc = upload(p, &p->d.images, imgs.data(), imgs.size());
    if (rc == RF_OK) rc = upload(p, &p->d.blocks, blocks.data(), blocks.size());
    if (rc == RF_OK) rc = upload(p, &p->d.blocks2, blocks2.data(), blocks2.size());
    if (rc == RF_OK) RF_CUDA_CHECK(cudaStreamSynchronize(p->tab_stream));
    return rc;
}

}  // namespace rf
