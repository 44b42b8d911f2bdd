// rf_internal.h -- plan object and internal interfaces of librealfast_b200 (not installed).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "../../include/realfast.h"

namespace rf {

void set_error(const char* fmt, ...);
#define RF_CUDA_CHECK(expr)                                                               \
    do {                                                                                  \
        cudaError_t e__ = (expr);                                                         \
        if (e__ != cudaSuccess) {                                                         \
            rf::set_error("%s failed: %s (%s:%d)", #expr, cudaGetErrorString(e__),        \
                          __FILE__, __LINE__);                                            \
            return RF_ERR_CUDA;                                                           \
        }                                                                                 \
    } while (0)

// uv columns gridded + transformed by one pass-1 CTA (bounded by its shared-memory tile)
inline int cols_per_group(int npix) { return npix <= 512 ? 16 : (npix == 1024 ? 8 : 4); }
constexpr int kWarpsPerCta = 8;     // 256 threads everywhere
constexpr int kThreads = 32 * kWarpsPerCta;
constexpr float kHistRange = 3.5f;  // histogram covers +-kHistRange * sigma_rms

// One image of the search loop: 16 bytes, device-resident list.
struct ImgDesc {
    int32_t dm_idx, dt_idx, j, dt;
};

// Gridding entry (8 bytes): one (baseline, channel) sample routed to one half-plane cell.
//   w0: bits 0..23  vis element  bl*nchan + ch
//       bits 24..28 distance (in lanes) to the first lane of the same cell in this 32-chunk
//       bit  29     last lane of its cell run inside the chunk (the lane that commits)
//       bit  30     conjugate (the sample enters through its Hermitian mirror)
//       bit  31     valid (0 = padding)
//   w1: bits 0..11  channel; bits 12..23 grid row (iv mod N); bits 24..27 column inside the group
struct GridEntry {
    uint32_t w0, w1;
};

struct DeviceTables {
    // integer tables (a), (c)
    int32_t* delay = nullptr;        // [ndm][nchan]
    int32_t* cell = nullptr;         // [nbl][nchan][2]
    uint8_t* keep = nullptr;         // [nbl][nchan]
    // gridding lists
    GridEntry* entries = nullptr;    // [n_chunks * 32]
    int32_t* warp_chunk = nullptr;   // [ngroups * kWarpsPerCta + 1] first chunk of each warp range
    ImgDesc* images = nullptr;       // [n_images]
    // plan inputs on device
    double* freqs = nullptr;         // [nchan] Hz
    double* uvw = nullptr;           // [nbl][3]
    double* dms = nullptr;           // [ndm]
    float2* twiddles = nullptr;      // [16 + 256] FFT stage twiddles
};

struct Workspace {
    float2* H = nullptr;             // [batch][npix][cpad] column-transformed half plane
    float* sumsq = nullptr;          // [batch][ngroups] Parseval partial sums of |G|^2 (weighted)
    uint32_t* hist = nullptr;        // [batch][nbins] merged histograms (row-split > 1)
    float* peak_val = nullptr;       // [batch][rsplit]
    int32_t* peak_pos = nullptr;     // [batch][rsplit]
    uint32_t* ticket = nullptr;      // [batch/2]
    int32_t* counters = nullptr;     // [4] device counters: stats_overflow, ...
    ImgDesc* dbg_desc = nullptr;     // one descriptor for rf_debug_image
    int batch = 0, rsplit = 1;
    size_t h_elems = 0;
};

}  // namespace rf

struct rf_plan {
    int nchan = 0, nbl = 0, npol = 0, nint = 0, npix = 0, ndm = 0, ndt = 0;
    double inttime = 0, cell = 0;
    float threshold = 0;
    int span = 0;                    // streaming search span (0 = all valid)
    int user_batch = 0;
    std::vector<double> freqs, uvw, dms;
    std::vector<int32_t> dts;
    std::vector<float> weights;      // [nchan]
    // host copies of the tables
    std::vector<int32_t> h_delay, h_cell;
    std::vector<uint8_t> h_keep;
    std::vector<int32_t> h_maxdelay;           // [ndm]
    std::vector<int32_t> h_num_t;              // [ndm][ndt]
    // derived
    int n_kept = 0, n_dropped = 0;
    int ncol = 0;                    // occupied half-plane columns 0..ncol-1 (ncol <= npix/2+1)
    int colgrp = 16;                 // columns per pass-1 CTA = rf::cols_per_group(npix)
    int cpad = 0;                    // ncol rounded up to colgrp
    int ngroups = 0;
    int nbins = 2048;
    int64_t n_images = 0, vis_gridded = 0;
    int64_t n_entries = 0, n_chunks = 0;
    int last_launches = 0;
    // rf_search_host staging
    void* stage_vis = nullptr;
    rf_cand* stage_cand = nullptr;
    int32_t* stage_count = nullptr;
    int stage_capacity = 0;
    cudaStream_t own_stream = nullptr;
    // per-kernel event timing
    bool profile = false;
    std::vector<cudaEvent_t> events;
    int n_events_used = 0;
    rf::DeviceTables d;
    rf::Workspace ws;
};

namespace rf {
// rf_tables.cu
int build_delay_table(rf_plan* p);            // device kernel (float64) -> d.delay, h_delay
int build_cell_table(rf_plan* p);             // device kernel (float64) -> d.cell/keep, host copies
int build_grid_lists(rf_plan* p);             // host binning of the cell table -> d.entries, d.warp_chunk
int build_image_list(rf_plan* p);             // (dm, dt, j) loop -> d.images
// rf_search.cu
int ensure_workspace(rf_plan* p);
void free_workspace(rf_plan* p);
int launch_search(rf_plan* p, const void* vis, cudaStream_t st, rf_cand_out* out);
int launch_debug_image(rf_plan* p, const void* vis, int dm_idx, int dt_idx, int t_idx,
                       float* image_dev, rf_cand* stats_dev, cudaStream_t st);
}  // namespace rf
