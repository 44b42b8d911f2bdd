// rf_api.cu -- the C-ABI of include/realfast.h: validation, plan lifetime, error strings.
#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>

#include "rf_internal.h"

namespace rf {
static thread_local char g_err[512] = "";
void set_error(const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}
}  // namespace rf

using rf::set_error;

namespace {

bool finite_pos(double x) { return std::isfinite(x) && x > 0.0; }

int rebuild_geometry(rf_plan* p) {
    int rc;
    if ((rc = rf::build_cell_table(p)) != RF_OK) return rc;
    if ((rc = rf::build_grid_lists(p)) != RF_OK) return rc;
    if ((rc = rf::build_image_list(p)) != RF_OK) return rc;   // vis_gridded depends on N_w
    return RF_OK;
}

// A plan lives on the device it was created on (tables, workspace, kernel attributes): the caller must have that
// device current when it enqueues work.
int check_device(const rf_plan* p) {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != p->device) {
        set_error("plan was created on CUDA device %d but device %d is current", p->device, dev);
        return RF_ERR_STATE;
    }
    return RF_OK;
}

void free_tables(rf_plan* p) {
    rf::DeviceTables& d = p->d;
    cudaFree(d.delay); cudaFree(d.cell); cudaFree(d.keep); cudaFree(d.gen.entries); cudaFree(d.gen.warp_chunk);
    cudaFree(d.tree.entries); cudaFree(d.tree.cells); cudaFree(d.tree.stream_iter); cudaFree(d.tree.stream_cell); cudaFree(d.tree.group_cell); cudaFree(d.tree.dft_blk); cudaFree(d.tree.dft_off); cudaFree(d.blocks); cudaFree(d.blocks2);
    for (uint2* e : d.aux_entries) cudaFree(e); cudaFree(d.images); cudaFree(d.freqs); cudaFree(d.uvw); cudaFree(d.dms); cudaFree(d.weights); cudaFree(d.twiddles); cudaFree(d.twp);
    p->dev_cap.clear();
    d = rf::DeviceTables{};
}

}  // namespace

extern "C" {

const char* rf_last_error(void) { return rf::g_err; }

int rf_plan_create(rf_plan** out, const double* freqs_hz, int nchan, const double* uvw_m, int nbl,
                   int npol, int nint, double inttime_s, int npix, double cell_rad,
                   const double* dm_list, int ndm, const int32_t* dt_list, int ndt,
                   float threshold_sigma) {
    if (out) *out = nullptr;
    if (!out || !freqs_hz || !uvw_m || !dm_list || !dt_list) { set_error("null pointer argument"); return RF_ERR_ARG; }
    if (nchan <= 0 || nbl <= 0 || nint <= 0 || ndm <= 0 || ndt <= 0) { set_error("counts must be positive"); return RF_ERR_ARG; }
    if (nchan > 4096) { set_error("nchan %d > 4096", nchan); return RF_ERR_ARG; }
    if ((long long)nbl * nchan >= (1ll << 24)) { set_error("nbl*nchan must be < 2^24"); return RF_ERR_ARG; }
    if (nbl >= (1 << 16)) { set_error("nbl must be < 2^16"); return RF_ERR_ARG; }
    if (npol != 1 && npol != 2 && npol != 4) { set_error("npol must be 1, 2 or 4"); return RF_ERR_ARG; }
    if (npix < 64 || npix > 4096 || (npix & (npix - 1))) { set_error("npix must be a power of two in 64..4096"); return RF_ERR_ARG; }
    if (!finite_pos(inttime_s) || !finite_pos(cell_rad)) { set_error("inttime and cell must be finite and positive"); return RF_ERR_ARG; }
    if (!std::isfinite(threshold_sigma)) { set_error("threshold must be finite"); return RF_ERR_ARG; }
    for (int i = 0; i < nchan; i++) if (!finite_pos(freqs_hz[i])) { set_error("freqs_hz[%d] not finite/positive", i); return RF_ERR_ARG; }
    for (int i = 0; i < 3 * nbl; i++) if (!std::isfinite(uvw_m[i])) { set_error("uvw_m[%d] not finite", i); return RF_ERR_ARG; }
    for (int i = 0; i < ndm; i++) if (!std::isfinite(dm_list[i]) || dm_list[i] < 0) { set_error("dm_list[%d] must be finite and >= 0", i); return RF_ERR_ARG; }
    for (int i = 0; i < ndt; i++) if (dt_list[i] <= 0) { set_error("dt_list[%d] must be >= 1", i); return RF_ERR_ARG; }

    rf_plan* p = new (std::nothrow) rf_plan();
    if (!p) { set_error("host allocation failed"); return RF_ERR_NOMEM; }
    p->nchan = nchan; p->nbl = nbl; p->npol = npol; p->nint = nint; p->npix = npix;
    p->ndm = ndm; p->ndt = ndt; p->inttime = inttime_s; p->cell = cell_rad; p->threshold = threshold_sigma;
    p->freqs.assign(freqs_hz, freqs_hz + nchan);
    p->uvw.assign(uvw_m, uvw_m + 3 * (size_t)nbl);
    p->dms.assign(dm_list, dm_list + ndm);
    p->dts.assign(dt_list, dt_list + ndt);
    p->weights.assign(nchan, 1.0f);
    p->nbins = 2048;
    rf::configure_tree(p);
    if (cudaGetDevice(&p->device) != cudaSuccess) {
        set_error("cudaGetDevice failed: %s", cudaGetErrorString(cudaGetLastError()));
        delete p;
        return RF_ERR_CUDA;
    }
    if (cudaStreamCreateWithFlags(&p->tab_stream, cudaStreamNonBlocking) != cudaSuccess) {
        set_error("cudaStreamCreate failed: %s", cudaGetErrorString(cudaGetLastError()));
        delete p;
        return RF_ERR_CUDA;
    }
    int rc = rf::build_delay_table(p);
    if (rc == RF_OK) rc = rebuild_geometry(p);
    if (rc != RF_OK) { rf_plan_destroy(p); return rc; }
    *out = p;
    return RF_OK;
}

int rf_plan_destroy(rf_plan* p) {
    if (!p) return RF_OK;
    for (cudaEvent_t e : p->events) cudaEventDestroy(e);
    cudaFree(p->stage_vis); cudaFree(p->stage_cand); cudaFree(p->stage_count);
    if (p->own_stream) cudaStreamDestroy(p->own_stream);
    if (p->copy_stream) cudaStreamDestroy(p->copy_stream);
    for (cudaEvent_t e : p->chunk_done) cudaEventDestroy(e);
    if (p->tab_stream) cudaStreamDestroy(p->tab_stream);
    rf::free_workspace(p);
    free_tables(p);
    delete p;
    return RF_OK;
}

int rf_search(rf_plan* p, const void* vis_dev, void* cuda_stream, rf_cand_out* out) {
    if (!p || !vis_dev || !out || !out->count || (out->capacity > 0 && !out->items) || out->capacity < 0) {
        set_error("null pointer argument");
        return RF_ERR_ARG;
    }
    if (reinterpret_cast<uintptr_t>(vis_dev) & 15) { set_error("vis_dev must be 16-byte aligned"); return RF_ERR_ARG; }
    if (int rc_d = check_device(p)) return rc_d;
    return rf::launch_search(p, vis_dev, static_cast<cudaStream_t>(cuda_stream), out);
}

int rf_search_host(rf_plan* p, const void* vis_host, rf_cand* cand_host, int32_t capacity, int32_t* count_host) {
    if (!p || !vis_host || !count_host || capacity < 0 || (capacity > 0 && !cand_host)) {
        set_error("null pointer argument");
        return RF_ERR_ARG;
    }
    if (int rc_d = check_device(p)) return rc_d;
    const size_t vis_bytes = (size_t)p->nint * p->nbl * p->nchan * p->npol * 8;
    if (!p->own_stream) RF_CUDA_CHECK(cudaStreamCreateWithFlags(&p->own_stream, cudaStreamNonBlocking));
    if (!p->stage_vis) RF_CUDA_CHECK(cudaMalloc(&p->stage_vis, vis_bytes));
    if (!p->stage_count) RF_CUDA_CHECK(cudaMalloc((void**)&p->stage_count, sizeof(int32_t)));
    if (p->stage_capacity < capacity || !p->stage_cand) {
        cudaFree(p->stage_cand);
        p->stage_cand = nullptr;
        RF_CUDA_CHECK(cudaMalloc((void**)&p->stage_cand, (size_t)(capacity > 0 ? capacity : 1) * sizeof(rf_cand)));
        p->stage_capacity = capacity;
    }
    cudaStream_t st = p->own_stream;
    rf_cand_out out{p->stage_cand, capacity, p->stage_count};
    int rc;
    if (p->tree_tb > 0 && p->n_blocks > 0 && !p->meansub && p->n_kept > 0) {
        // The boxcar-tree search consumes the segment front to back: upload it in chunks on a copy stream and
        // let the search run behind the upload (each launch waits only for the integrations it reads).
        const int rows = 64;       // chunks of 32 integrations measured the same end to end (43.3 vs 43.3 ms at L-band), 128: 45.0 ms
        const int n_chunks = (p->nint + rows - 1) / rows;
        if (!p->copy_stream) RF_CUDA_CHECK(cudaStreamCreateWithFlags(&p->copy_stream, cudaStreamNonBlocking));
        while ((int)p->chunk_done.size() < n_chunks) {
            cudaEvent_t e;
            RF_CUDA_CHECK(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
            p->chunk_done.push_back(e);
        }
        const size_t row_bytes = (size_t)p->nbl * p->nchan * p->npol * 8;
        for (int c = 0; c < n_chunks; c++) {
            const size_t lo = (size_t)c * rows, hi = std::min<size_t>(p->nint, lo + rows);
            RF_CUDA_CHECK(cudaMemcpyAsync(static_cast<char*>(p->stage_vis) + lo * row_bytes,
                                          static_cast<const char*>(vis_host) + lo * row_bytes, (hi - lo) * row_bytes,
                                          cudaMemcpyHostToDevice, p->copy_stream));
            RF_CUDA_CHECK(cudaEventRecord(p->chunk_done[c], p->copy_stream));
        }
        rf::HostFeed feed{p->chunk_done.data(), rows, n_chunks};
        rc = rf::launch_search(p, p->stage_vis, st, &out, &feed);
        if (rc != RF_OK) { cudaStreamSynchronize(p->copy_stream); return rc; }
    } else {
        RF_CUDA_CHECK(cudaMemcpyAsync(p->stage_vis, vis_host, vis_bytes, cudaMemcpyHostToDevice, st));
        rc = rf::launch_search(p, p->stage_vis, st, &out);
        if (rc != RF_OK) return rc;
    }
    RF_CUDA_CHECK(cudaMemcpyAsync(count_host, p->stage_count, sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    RF_CUDA_CHECK(cudaStreamSynchronize(st));
    const int32_t n = *count_host < capacity ? *count_host : capacity;
    if (n > 0) RF_CUDA_CHECK(cudaMemcpy(cand_host, p->stage_cand, (size_t)n * sizeof(rf_cand), cudaMemcpyDeviceToHost));
    return RF_OK;
}

int rf_plan_set_profiling(rf_plan* p, int enable) {
    if (!p) { set_error("null plan"); return RF_ERR_ARG; }
    p->profile = enable != 0;
    return RF_OK;
}

int rf_plan_get_kernel_times(rf_plan* p, float ms[4], int32_t launches[4]) {
    if (!p || !ms || !launches) { set_error("null pointer argument"); return RF_ERR_ARG; }
    for (int k = 0; k < 4; k++) { ms[k] = 0.f; launches[k] = 0; }
    for (int i = 1; i < p->n_events_used; i++) {
        const int kind = p->event_kind[i];
        if (kind < 0 || kind > 3) continue;
        float a = 0.f;
        RF_CUDA_CHECK(cudaEventElapsedTime(&a, p->events[i - 1], p->events[i]));
        ms[kind] += a;
        launches[kind]++;
    }
    return RF_OK;
}

int rf_plan_set_mode(rf_plan* p, int use_tree) {
    if (!p) { set_error("null plan"); return RF_ERR_ARG; }
    p->use_tree = use_tree != 0;
    rf::configure_tree(p);
    return rebuild_geometry(p);
}

int rf_plan_set_meansub(rf_plan* p, int enable) {
    if (!p) { set_error("null plan"); return RF_ERR_ARG; }
    p->meansub = enable != 0;
    return RF_OK;
}

int rf_prep_meansub(rf_plan* p, void* vis_dev, void* cuda_stream) {
    if (!p || !vis_dev) { set_error("null pointer argument"); return RF_ERR_ARG; }
    if (reinterpret_cast<uintptr_t>(vis_dev) & 15) { set_error("vis_dev must be 16-byte aligned"); return RF_ERR_ARG; }
    if (int rc_d = check_device(p)) return rc_d;
    return rf::launch_meansub_inplace(p, vis_dev, static_cast<cudaStream_t>(cuda_stream));
}

int rf_plan_set_chan_weights(rf_plan* p, const float* w) {
    if (!p || !w) { set_error("null pointer argument"); return RF_ERR_ARG; }
    for (int i = 0; i < p->nchan; i++) p->weights[i] = (w[i] != 0.0f) ? 1.0f : 0.0f;
    return rebuild_geometry(p);
}

int rf_plan_set_uvw(rf_plan* p, const double* uvw_m, double cell_rad) {
    if (!p || !uvw_m) { set_error("null pointer argument"); return RF_ERR_ARG; }
    for (int i = 0; i < 3 * p->nbl; i++) if (!std::isfinite(uvw_m[i])) { set_error("uvw_m[%d] not finite", i); return RF_ERR_ARG; }
    if (cell_rad > 0) {
        if (!std::isfinite(cell_rad)) { set_error("cell must be finite"); return RF_ERR_ARG; }
        p->cell = cell_rad;
    }
    p->uvw.assign(uvw_m, uvw_m + 3 * (size_t)p->nbl);
    return rebuild_geometry(p);
}

int rf_plan_set_search_span(rf_plan* p, int n) {
    if (!p || n < 0) { set_error("invalid span"); return RF_ERR_ARG; }
    p->span = n;
    return rf::build_image_list(p);
}

int rf_plan_set_batch(rf_plan* p, int n) {
    if (!p || n < 0) { set_error("invalid batch"); return RF_ERR_ARG; }
    p->user_batch = n;
    return RF_OK;
}

int rf_plan_set_tuning(rf_plan* p, int knob, int value) {
    if (!p) { set_error("null plan"); return RF_ERR_ARG; }
    switch (knob) {
        case RF_TUNE_AUX_WIDTHS: p->tune_aux = value != 0; break;
        case RF_TUNE_DM_GROUP:
            if (value < 1) { set_error("DM group must be >= 1"); return RF_ERR_ARG; }
            p->tune_dm_group = value;
            break;
        case RF_TUNE_FEED_BATCH:
            if (value < 0) { set_error("feed batch must be >= 0"); return RF_ERR_ARG; }
            p->tune_feed_batch = value;
            return RF_OK;                              // read at launch time: nothing to rebuild
        case RF_TUNE_TREE_MAXPIX:
            if (value < 0) { set_error("tree maxpix must be >= 0"); return RF_ERR_ARG; }
            p->tune_tree_maxpix = value;
            break;
        case RF_TUNE_GATHER_ORDER:
            p->tune_gather_order = value != 0;
            return RF_OK;
        case RF_TUNE_COL_DFT:
            if (value < 0 || value > rf::kDftMaxSpc) { set_error("blocks per column-pass CTA must be in 0..%d", rf::kDftMaxSpc); return RF_ERR_ARG; }
            p->tune_col_dft = value;
            return RF_OK;
        default: set_error("unknown tuning knob %d", knob); return RF_ERR_ARG;
    }
    rf::configure_tree(p);
    return rebuild_geometry(p);
}

int rf_plan_get_tables(rf_plan* p, int32_t* delay_host, int32_t* cell_host, uint8_t* keep_host) {
    if (!p) { set_error("null plan"); return RF_ERR_ARG; }
    if (delay_host) memcpy(delay_host, p->h_delay.data(), p->h_delay.size() * sizeof(int32_t));
    if (cell_host) memcpy(cell_host, p->h_cell.data(), p->h_cell.size() * sizeof(int32_t));
    if (keep_host) memcpy(keep_host, p->h_keep.data(), p->h_keep.size());
    return RF_OK;
}

int64_t rf_plan_num_images(const rf_plan* p) { return p ? p->n_images : 0; }

int rf_plan_fft_work(const rf_plan* p, int64_t* col_transforms, int64_t* row_transforms) {
    if (!p) { set_error("null plan"); return RF_ERR_ARG; }
    if (col_transforms) *col_transforms = p->n_col_fft;
    if (row_transforms) *row_transforms = p->n_row_fft;
    return RF_OK;
}

int rf_plan_num_t(const rf_plan* p, int dm_idx, int dt_idx) {
    if (!p || dm_idx < 0 || dm_idx >= p->ndm || dt_idx < 0 || dt_idx >= p->ndt) return RF_ERR_ARG;
    return p->h_num_t[(size_t)dm_idx * p->ndt + dt_idx];
}

int rf_debug_image(rf_plan* p, const void* vis_dev, int dm_idx, int dt_idx, int t_idx,
                   float* image_dev, rf_cand* stats_dev, void* cuda_stream) {
    if (!p || !vis_dev) { set_error("null pointer argument"); return RF_ERR_ARG; }
    if (dm_idx < 0 || dm_idx >= p->ndm || dt_idx < 0 || dt_idx >= p->ndt) { set_error("trial index out of range"); return RF_ERR_STATE; }
    const int dt = p->dts[dt_idx];
    if (t_idx < 0 || (long long)(t_idx + 1) * dt > p->nint - p->h_maxdelay[dm_idx]) { set_error("t_idx out of range"); return RF_ERR_STATE; }
    if (int rc_d = check_device(p)) return rc_d;
    return rf::launch_debug_image(p, vis_dev, dm_idx, dt_idx, t_idx, image_dev, stats_dev,
                                  static_cast<cudaStream_t>(cuda_stream));
}

int rf_cand_spectrum(rf_plan* p, const void* vis_dev, int dm_idx, int dt_idx, int t_idx, int l_pix, int m_pix,
                     int half_window, float* spec_dev, void* cuda_stream) {
    if (!p || !vis_dev || !spec_dev) { set_error("null pointer argument"); return RF_ERR_ARG; }
    if (dm_idx < 0 || dm_idx >= p->ndm || dt_idx < 0 || dt_idx >= p->ndt) { set_error("trial index out of range"); return RF_ERR_STATE; }
    if (half_window < 0 || half_window > 32767) { set_error("half_window out of range"); return RF_ERR_ARG; }
    if (l_pix < -p->npix || l_pix >= p->npix || m_pix < -p->npix || m_pix >= p->npix) { set_error("pixel out of range"); return RF_ERR_ARG; }
    if (int rc_d = check_device(p)) return rc_d;
    return rf::launch_cand_spectrum(p, vis_dev, dm_idx, dt_idx, t_idx, l_pix, m_pix, half_window, spec_dev,
                                    static_cast<cudaStream_t>(cuda_stream));
}

int rf_inject(rf_plan* p, void* vis_dev, double amp, double l_pix, double m_pix, double dm, int width, int t0,
              void* cuda_stream) {
    if (!p || !vis_dev) { set_error("null pointer argument"); return RF_ERR_ARG; }
    if (!std::isfinite(amp) || !std::isfinite(l_pix) || !std::isfinite(m_pix) || !std::isfinite(dm) || dm < 0 || width < 0) {
        set_error("invalid source parameters");
        return RF_ERR_ARG;
    }
    if (int rc_d = check_device(p)) return rc_d;
    return rf::launch_inject(p, vis_dev, amp, l_pix, m_pix, dm, width, t0, static_cast<cudaStream_t>(cuda_stream));
}

int rf_search_periodic(rf_plan* p, const void* vis_dev, void* cuda_stream, rf_cand_out* out) {
    if (!p || !vis_dev || !out || !out->count || (out->capacity > 0 && !out->items) || out->capacity < 0) {
        set_error("null pointer argument");
        return RF_ERR_ARG;
    }
    if (reinterpret_cast<uintptr_t>(vis_dev) & 15) { set_error("vis_dev must be 16-byte aligned"); return RF_ERR_ARG; }
    if (int rc_d = check_device(p)) return rc_d;
    return rf::launch_search_periodic(p, vis_dev, static_cast<cudaStream_t>(cuda_stream), out, -1, 0, nullptr, nullptr);
}

int rf_plan_periodic_nt(const rf_plan* p, int dm_idx) {
    if (!p || dm_idx < 0 || dm_idx >= p->ndm) return RF_ERR_ARG;
    return rf::periodic_nt(p, dm_idx);
}

int rf_debug_periodic_image(rf_plan* p, const void* vis_dev, int dm_idx, int k, float* power_dev, rf_cand* stats_dev,
                            void* cuda_stream) {
    if (!p || !vis_dev) { set_error("null pointer argument"); return RF_ERR_ARG; }
    if (dm_idx < 0 || dm_idx >= p->ndm) { set_error("trial index out of range"); return RF_ERR_STATE; }
    const int nt = rf::periodic_nt(p, dm_idx);
    if (k < 1 || k > nt / 2) { set_error("fluctuation-frequency bin out of range"); return RF_ERR_STATE; }
    if (int rc_d = check_device(p)) return rc_d;
    return rf::launch_search_periodic(p, vis_dev, static_cast<cudaStream_t>(cuda_stream), nullptr, dm_idx, k, power_dev,
                                      stats_dev);
}

int rf_plan_get_counters(rf_plan* p, rf_counters* out) {
    if (!p || !out) { set_error("null pointer argument"); return RF_ERR_ARG; }
    int32_t c[4] = {0, 0, 0, 0};
    if (p->ws.counters) RF_CUDA_CHECK(cudaMemcpy(c, p->ws.counters, sizeof(c), cudaMemcpyDeviceToHost));
    out->images = c[1];               // counted by the kernels: one per finalised image of the last search
    out->vis_gridded = p->vis_gridded;
    out->n_kept = p->n_kept;
    out->n_dropped = p->n_dropped;
    out->stats_overflow = c[0];
    out->kernel_launches = p->last_launches;
    return RF_OK;
}

}  // extern "C"
