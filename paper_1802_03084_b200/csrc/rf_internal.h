// rf_internal.h -- plan object and internal interfaces of librealfast_b200 (not installed).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <map>
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
constexpr int kDmGroup = 8;         // DM trials interleaved in time by the tree path's block order
constexpr size_t kSlidingSumBudget = (size_t)24 << 30;   // bytes of sliding-sum arrays (widths off the tree) per plan
constexpr int kUnitBlocks = 4;      // consecutive time blocks of a DM group kept together in the tree path's block order
constexpr int kGatherBlocks = 2;    // consecutive time blocks of one DM served by one gather CTA (adjacent in every block list);
                                    // 4 was measured no faster (L-band gather 5.69 vs 5.68 ms, S-band 209 vs 205 ms) and pads more
static_assert(kUnitBlocks % kGatherBlocks == 0, "a unit of the block order holds whole gather groups");
constexpr int kTreeUnroll = 8;      // iterations of the tree gather kept in flight per warp
constexpr int kStreamIters = 256;   // target length of one warp stream of the tree gather.  Measured (gather per step, L-band /
                                    // S-band, streams sorted by length): 32: 5.86 ms / 189 ms, 64: 5.19 / 164, 128: 4.77 / 150,
                                    // 256: 4.63 / 143, 512: 4.77 / 139 -- a CTA's set-up and pipeline fill amortise over its streams
constexpr float kHistRange = 3.5f;  // histogram covers +-kHistRange * sigma_rms (B1)

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

// One block of the image-domain boxcar tree: TB consecutive native integrations of one DM.
struct BlockDesc {
    int32_t dm_idx, tb, nsearch, pad;
};

// Tree-path gather entry (8 bytes): one (baseline, channel) sample of one half-plane cell.
//   x: (baseline * nchan + channel) * tpitch = offset of the sample's time series in visI (< 2^32, checked);
//      padding entries point at the all-zero series that follows the last one
//   y: bits 0..11 channel (for its delay); bit 28 EDGE: the cell lies on column 0 or N/2 (Parseval
//   weight 1 instead of 2); bit 29 END: last iteration of its cell (every entry of that iteration
//   carries it); bit 31 conjugate (= the sign bit of the imaginary part).
// Tree-path cell (4 bytes): bits 0..11 grid row; bits 12..15 column inside its column group;
//   bit 16: the cell lies on column 0 or N/2 (Parseval weight 1 instead of 2).
// Half-plane gridding lists for one choice of columns-per-CTA.
struct GridLists {
    GridEntry* entries = nullptr;    // device [n_chunks * 32]
    int32_t* warp_chunk = nullptr;   // device [ngroups * kWarpsPerCta + 1]
    int colgrp = 0, cpad = 0, ngroups = 0;
    int64_t n_chunks = 0;
};

// Work lists of the boxcar-tree path (built by build_grid_lists, see rf_tables.cu).
struct TreeLists {
    uint2* entries = nullptr;        // device [n_iters * lg]
    int32_t* stream_iter = nullptr;  // device [n_streams][2] iteration range of each warp stream, longest streams first
    int32_t* stream_cell = nullptr;  // device [n_streams] first cell of each warp stream
    uint32_t* cells = nullptr;       // device [n_cells] sorted by (column, row mod 16, row)
    int32_t* group_cell = nullptr;   // device [ngroups + 1] first cell of each column group
    int colgrp = 0, cpad = 0, ngroups = 0, lg = 0;
    int n_cells = 0, n_streams = 0, n_parts = 0;   // n_parts = gather CTAs per block
    int max_group_cells = 0;         // most cells in one column group
    int32_t* dft_blk = nullptr;      // device, npix >= 2048: list blocks of k_tree_coldft, one per column group
    int32_t* dft_off = nullptr;      // device [ngroups + 1] first int of each block
    int dft_max_blk = 0;             // ints in the longest block
    int64_t n_iters = 0;
};

struct DeviceTables {
    // integer tables (a), (c)
    int32_t* delay = nullptr;        // [ndm][nchan]
    int32_t* cell = nullptr;         // [nbl][nchan][2]
    uint8_t* keep = nullptr;         // [nbl][nchan]
    // gridding lists: generic path (colgrp = cols_per_group) and boxcar-tree path
    GridLists gen;
    TreeLists tree;
    std::vector<uint2*> aux_entries; // [ndt] gather entries of a width off the tree: tree.entries with the row pitch of its
                                     // phase-decimated sum array (null = width not searched that way); sized once
    BlockDesc* blocks2 = nullptr;    // their blocks, all such widths one after the other (rf_plan::aux_first)
    ImgDesc* images = nullptr;       // [n_gen_images] images searched by the generic path
    BlockDesc* blocks = nullptr;     // [n_blocks] blocks searched by the tree path
    // plan inputs on device
    double* freqs = nullptr;         // [nchan] Hz
    double* uvw = nullptr;           // [nbl][3]
    double* dms = nullptr;           // [ndm]
    float* weights = nullptr;        // [nchan]
    float2* twiddles = nullptr;      // [16 + 256] FFT stage twiddles
    float2* twp = nullptr;           // [16][15] stage-2 twiddle powers
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
    size_t cap_H = 0, cap_sumsq = 0, cap_hist = 0, cap_peak_val = 0, cap_peak_pos = 0, cap_ticket = 0;   // elements
    // boxcar-tree path
    float2* visI = nullptr;          // [nbl*nchan][tpitch] Stokes-I (pol sum), time fastest
    float2* Ht = nullptr;            // [blk_batch][npix][cpad_tree][TB]
    float* sumsq_t = nullptr;        // [blk_batch][2*TB-1][n_parts] Parseval partials of the gather CTAs
    float2* cellsum = nullptr;       // [blk_batch][n_cells][TB] gridded cell sums (compact grid)
    BlockDesc* dbg_block = nullptr;
    int blk_batch = 0;
    size_t visI_elems = 0, ht_elems = 0, cs_elems = 0, ss_elems = 0;
    float2* visS = nullptr;          // phase-decimated boxcar sums of the widths off the tree (B7), one array per width
    std::vector<size_t> aux_off;     // [ndt + 1] first element of each width's array in visS
    size_t visS_elems = 0;
    // periodicity search
    float2* slab = nullptr;          // [n_slabs][nbl*nchan][slab_pitch] time spectra as (S, -i S) pairs
    size_t slab_elems = 0;
    int n_slabs = 0, slab_pitch = 0;
    BlockDesc* pblocks = nullptr;    // block list of the periodicity search
    std::vector<BlockDesc> h_pblocks; // its host copy (re-uploaded only when it changes)
    size_t pblocks_cap = 0;
    int32_t* zero_delay = nullptr;   // [nchan] zeros: the slabs are already dedispersed
    float2* time_tw = nullptr;       // [7][16 + 256] twiddles of the time transforms, NT = 64 << i
    // prep (mean-visibility subtraction)
    double2* mean_partial = nullptr; // [kMeanChunks][nbl*nchan*npol]
    float2* mean_p = nullptr;        // [nbl*nchan*npol] time mean per polarisation product
    float2* mean_i = nullptr;        // [nbl*nchan] sum over pol of mean_p
};

}  // namespace rf

struct rf_plan {
    int nchan = 0, nbl = 0, npol = 0, nint = 0, npix = 0, ndm = 0, ndt = 0;
    double inttime = 0, cell = 0;
    float threshold = 0;
    int span = 0;                    // streaming search span (0 = all valid)
    bool use_tree = true;            // image-domain boxcar tree for power-of-two dt (rf_plan_set_mode)
    bool meansub = false;            // search vis - mean_t(vis) (rf_plan_set_meansub)
    int user_batch = 0;
    int device = 0;                  // CUDA device the plan was created on (checked by every entry point that launches)
    // tuning knobs (rf_plan_set_tuning): none of them changes a result
    bool tune_aux = true;            // widths off the tree ride the tree kernels on phase-decimated sums (B7)
    int tune_dm_group = rf::kDmGroup;   // DM trials interleaved in time by the block order
    int tune_feed_batch = 0;         // blocks per launch behind an upload (0 = two waves of row-pass CTAs)
    int tune_tree_maxpix = 4096;     // largest npix searched by the boxcar-tree kernels
    int tune_col_dft = 6;            // npix >= 2048: column pass as a pruned DFT over the occupied cells (k_tree_coldft), a CTA
                                     // keeps one column group for this many blocks of a launch; 0 = column FFTs
    int tune_gather_order = 1;       // 1 = gather grid runs over block pairs fastest (cell-range major), 0 = cell ranges fastest
    std::map<const void*, size_t> smem_attr;   // dynamic shared memory opted in per kernel, on this plan's device
    std::vector<double> freqs, uvw, dms;
    std::vector<int32_t> dts;
    std::vector<float> weights;      // [nchan]
    // host copies of the tables
    std::vector<int32_t> h_delay, h_cell;
    std::vector<uint8_t> h_keep;
    std::vector<int32_t> h_maxdelay;           // [ndm]
    std::vector<int32_t> h_num_t;              // [ndm][ndt]
    std::vector<int32_t> aux_width;            // [ndt] 1 = width off the tree searched by the tree kernels on its phase-decimated sums
    std::vector<int32_t> aux_pitch;            // [ndt] row pitch of that array (output integrations per series and phase)
    std::vector<int64_t> aux_first;            // [ndt + 1] first block of each width in d.blocks2
    std::vector<int32_t> h_block_deadline;     // [n_blocks] integrations [0, deadline) are all a tree block (and those before it) read
    // derived
    int n_kept = 0, n_dropped = 0;
    int ncol = 0;                    // occupied half-plane columns 0..ncol-1 (ncol <= npix/2+1)
    // boxcar tree (image-domain resampling): TB = largest power-of-two dt handled by the tree
    // (0 = tree path off); level l <-> dt = 2^l; tree_dt_idx[l] = index in dt_list or -1
    int tree_tb = 0;
    int tree_dt_idx[4] = {-1, -1, -1, -1};
    int tpitch = 0;                  // time pitch of visI (>= nint + TB, multiple of 16)
    int64_t n_blocks = 0, n_gen_images = 0;
    int nbins = 2048;
    int64_t n_images = 0, vis_gridded = 0;
    int64_t n_col_fft = 0, n_row_fft = 0;      // npix-point transforms one rf_search runs (column pass; row pass = pair transforms)
    int64_t n_entries = 0;
    int last_launches = 0;
    // rf_search_host staging
    void* stage_vis = nullptr;
    rf_cand* stage_cand = nullptr;
    int32_t* stage_count = nullptr;
    int stage_capacity = 0;
    cudaStream_t own_stream = nullptr, copy_stream = nullptr;
    std::vector<cudaEvent_t> chunk_done;       // upload events of rf_search_host
    // per-kernel event timing
    bool profile = false;
    std::vector<cudaEvent_t> events;
    std::vector<int> event_kind;
    int n_events_used = 0;
    rf::DeviceTables d;
    std::map<void*, size_t> dev_cap;   // capacity in bytes of each table pointer (rf_tables.cu)
    cudaStream_t tab_stream = nullptr; // plan-time kernels and table copies (non-blocking)
    rf::Workspace ws;
};

namespace rf {
// rf_tables.cu
int build_delay_table(rf_plan* p);            // device kernel (float64) -> d.delay, h_delay
int build_cell_table(rf_plan* p);             // device kernel (float64) -> d.cell/keep, host copies
int build_grid_lists(rf_plan* p);             // host binning of the cell table -> d.gen, d.tree
int aux_pitch_of(const rf_plan* p, int dt);   // row pitch of the phase-decimated sum array of a width
int build_image_list(rf_plan* p);             // (dm, dt, j) loop -> d.images (generic) + d.blocks (tree)
size_t phase_sum_smem(int dt, int* jc_out);   // dynamic shared memory (and JC) of k_phase_sum for a width
constexpr int kDftMaxSpc = 64;        // k_tree_coldft: most blocks of a launch one CTA walks (RF_TUNE_COL_DFT)
constexpr size_t kMaxDynSmem = 227 * 1024;    // opt-in limit per CTA on sm_100a
// cudaFuncSetAttribute(MaxDynamicSharedMemorySize) once per (plan = device, kernel); kernels are per-device objects
int ensure_smem_attr(rf_plan* p, const void* kern, size_t smem);
int tree_cols_per_group(int npix, int tb);
void configure_tree(rf_plan* p);              // which dt values ride the boxcar tree    // columns per pass-1 CTA of the tree path
// rf_prep.cu
int launch_time_mean(rf_plan* p, const void* vis, cudaStream_t st);
int launch_meansub_inplace(rf_plan* p, void* vis, cudaStream_t st);
// rf_cutout.cu
int launch_cand_spectrum(rf_plan* p, const void* vis, int dm_idx, int dt_idx, int t_idx, int l_pix, int m_pix,
                         int half_window, float* spec_dev, cudaStream_t st);
int launch_inject(rf_plan* p, void* vis, double amp, double l_pix, double m_pix, double dm, int width, int t0,
                  cudaStream_t st);
// rf_search.cu
int ensure_workspace(rf_plan* p, bool need_generic);
void free_workspace(rf_plan* p);
// rf_search_host: the segment arrives in chunks of rows_per_chunk integrations (a multiple of 32); chunk c is
// on the device once chunk_done[c] has fired
struct HostFeed { const cudaEvent_t* chunk_done; int rows_per_chunk, n_chunks; };
int launch_search(rf_plan* p, const void* vis, cudaStream_t st, rf_cand_out* out, const HostFeed* feed = nullptr);
int launch_debug_image(rf_plan* p, const void* vis, int dm_idx, int dt_idx, int t_idx,
                       float* image_dev, rf_cand* stats_dev, cudaStream_t st);
int periodic_nt(const rf_plan* p, int dm_idx);   // length of the time transform of one DM trial (0 = none)
int launch_search_periodic(rf_plan* p, const void* vis, cudaStream_t st, rf_cand_out* out, int dbg_dm, int dbg_k,
                           float* power_dev, rf_cand* stats_dev);
}  // namespace rf
