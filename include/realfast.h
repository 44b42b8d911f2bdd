/* realfast.h -- C-ABI of the B200-native realfast search hot path.
 *
 * What the library computes (PAPER.md = Law et al., arXiv 1802.03084; readings
 * A1-A20 are listed in DESIGN.md):
 *
 *   for every DM trial x sampling time dt x output integration j of one segment
 *   of fast-sampled visibilities (the two dashed loops of Fig. 2):
 *     (a) shift each channel by its integer dispersion delay,
 *     (b) average dt integrations and the polarisations (Stokes I),
 *     (c) grid all baselines x channels on the uv plane, nearest cell, with the
 *         Hermitian conjugate,
 *     (d) form the image with a 2-D inverse FFT,
 *     (e) reduce it to peak, robust sigma and S/N and keep it if S/N >= threshold
 *         (PAPER.md:86-88).  An all-zero image (sigma = 0) has S/N := 0 and is never a
 *         candidate, whatever the threshold (reading A24).
 *
 * All device work is hand-written CUDA for sm_100a; there is no CPU fallback.
 * Every function returns RF_OK (0) or a negative error code, never throws, never
 * exits, never prints.  Unless said otherwise pointers are HOST pointers.
 */
#ifndef REALFAST_B200_H
#define REALFAST_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define RF_OK          0
#define RF_ERR_ARG    (-1)  /* null pointer, size out of range, non-finite value        */
#define RF_ERR_CUDA   (-2)  /* a CUDA runtime call failed; see rf_last_error()           */
#define RF_ERR_NOMEM  (-3)  /* host or device allocation failed                          */
#define RF_ERR_STATE  (-4)  /* call not valid for this plan (e.g. index out of range)    */

typedef struct rf_plan rf_plan;      /* opaque; owns all device tables and workspace */

/* One candidate: the image of (dm_idx, dt_idx, t_idx) had peak/sigma >= threshold.
 * t_idx is the index j in the dt-resampled series (native start = j * dt).
 * l_pix/m_pix are the signed pixel offsets of the peak in [-npix/2, npix/2): image
 * column x maps to l (via u), row y to m (via v); x >= npix/2 means x - npix (A12).  */
typedef struct {
    int32_t dm_idx, dt_idx, t_idx;
    int32_t l_pix, m_pix;
    float   peak, sigma, snr;
} rf_cand;                            /* 32 bytes */

/* Candidate sink, caller-owned DEVICE memory.  rf_search zeroes *count on the
 * stream before searching; count keeps counting past capacity (overflow = count >
 * capacity, extra candidates dropped).  Order of items is unspecified.          */
typedef struct {
    rf_cand* items;       /* device, capacity entries */
    int32_t  capacity;
    int32_t* count;       /* device, one int32 */
} rf_cand_out;

/* Counters of the last rf_search (read after synchronising its stream). */
typedef struct {
    int64_t images;           /* (dm, dt, j) images whose statistics the kernels finalised: counted ON
                                 THE DEVICE, once per image (rf_search_periodic: frequency images); equals
                                 rf_plan_num_images() after a complete rf_search, 0 when nothing is gridded */
    int64_t vis_gridded;      /* Stokes-I samples gridded = sum_images N_w * dt           */
    int32_t n_kept;           /* N_w: (baseline, channel) samples kept by the cell table  */
    int32_t n_dropped;        /* samples outside the grid or with zero channel weight      */
    int32_t stats_overflow;   /* images whose median/MAD fell outside the histogram range */
    int32_t kernel_launches;  /* kernels enqueued by the last rf_search                   */
} rf_counters;

/* Create a plan = the pipeline "state": everything that determines
 * the result except the visibilities.  All arrays are copied.
 *   freqs_hz [nchan]   channel centres, any order; delays are relative to max(freqs)
 *   uvw_m    [nbl][3]  baseline (u,v,w) in metres, one per segment; w is ignored
 *   npol               1, 2 or 4 polarisation products, averaged into Stokes I
 *   nint               integrations per segment; inttime_s seconds each
 *   npix               image side, power of two in 64..4096; cell_rad pixel size (rad)
 *   dm_list  [ndm]     pc/cm^3, any order; dt_list [ndt] widths >= 1 in integrations
 *   threshold_sigma    candidates have snr >= threshold (compared in float32)
 * Tables (a) delay[dm][ch] = floor(K DM (f^-2 - fmax^-2)/t_int + 0.5), K = 4.148808e-3
 * s GHz^2, and the uv cell table iu = floor(u f/c * npix*cell + 0.5) are computed on
 * the device in float64 and are bit-exact against the same expressions in IEEE-754.
 * Errors: RF_ERR_ARG on any invalid argument; RF_ERR_CUDA / RF_ERR_NOMEM.        */
int rf_plan_create(rf_plan** out,
                   const double* freqs_hz, int nchan,
                   const double* uvw_m, int nbl,
                   int npol, int nint, double inttime_s,
                   int npix, double cell_rad,
                   const double* dm_list, int ndm,
                   const int32_t* dt_list, int ndt,
                   float threshold_sigma);

/* Enqueue the whole search of one segment on `cuda_stream` (a cudaStream_t, may be
 * 0) and return without synchronising.  The device the plan was created on must be current
 * (RF_ERR_STATE otherwise; the same holds for every entry point that launches kernels).
 *   vis_dev  DEVICE pointer, complex64 [nint][nbl][nchan][npol] (re,im float32 pairs),
 *            16-byte aligned, borrowed read-only until the stream passes this work.
 * One rf_search in flight per plan (the workspace is per plan).                  */
int rf_search(rf_plan* plan, const void* vis_dev, void* cuda_stream, rf_cand_out* cand_out);

int rf_plan_destroy(rf_plan* plan);

/* Channel weights (0 = flagged: neither read nor counted in N_w; anything else = 1);
 * rebuilds the gridding tables (A17).  w [nchan] host floats.                     */
int rf_plan_set_chan_weights(rf_plan* plan, const float* w);

/* Replace the baseline uvw (and optionally the cell size: cell_rad <= 0 keeps it);
 * rebuilds the cell and gridding tables (hour angle changes between segments).
 * Deviation from SURVEY.md 8(b), which proposed (plan, uvw_m, cuda_stream): the cell size follows
 * max|uv| (reading A13) and so changes with uvw, and the rebuild sorts on the host, so it runs on the
 * plan's own non-blocking stream and returns when the tables are on the device; no caller stream is
 * involved.  The plan must be idle (no rf_search of it in flight).                              */
int rf_plan_set_uvw(rf_plan* plan, const double* uvw_m, double cell_rad);

/* Streaming (config 5): search only native integrations t < n_native_ints for every
 * DM (still bounded by nint - maxdelay(dm)); 0 restores "all valid" (A16).        */
int rf_plan_set_search_span(rf_plan* plan, int n_native_ints);

/* Copy the integer tables to HOST arrays (either may be NULL):
 *   delay_host [ndm][nchan]; cell_host [nbl][nchan][2] = (iu, iv) signed cells.
 *   keep_host [nbl][nchan] = 1 if the sample is gridded.                          */
int rf_plan_get_tables(rf_plan* plan, int32_t* delay_host, int32_t* cell_host, uint8_t* keep_host);

/* Number of images the plan searches, per rf_search; per (dm, dt) count via
 * rf_plan_num_t(plan, dm_idx, dt_idx).                                            */
int64_t rf_plan_num_images(const rf_plan* plan);
int     rf_plan_num_t(const rf_plan* plan, int dm_idx, int dt_idx);

/* Work accounting for the FFT rate (SURVEY.md 8(d) "secondary evidence"; the 2-D FFT is the paper's dominant
 * stage): the number of npix-point complex transforms ONE rf_search of this plan runs --
 * column pass (one per occupied-half-plane column, padded, per gridded integration) and row pass (one per image
 * row and PAIR of images: two real images share a complex transform).  Either pointer may be NULL.   */
int rf_plan_fft_work(const rf_plan* plan, int64_t* col_transforms, int64_t* row_transforms);

/* Pixel-parity hook: write the float32 image [npix][npix] (row y, column x, no
 * fftshift) of one (dm_idx, dt_idx, t_idx) to DEVICE memory, and optionally its
 * statistics (peak, sigma, snr as the search computes them) to a device rf_cand.
 * Runs the same kernels as rf_search.  Debug hook: may synchronise the stream.     */
int rf_debug_image(rf_plan* plan, const void* vis_dev, int dm_idx, int dt_idx, int t_idx,
                   float* image_dev, rf_cand* stats_dev, void* cuda_stream);

/* Counters of the most recent rf_search on this plan; synchronises nothing: call
 * after the caller has synchronised the stream.                                   */
int rf_plan_get_counters(rf_plan* plan, rf_counters* out);

/* Tuning knob (not part of the result): images per batch of the two-pass pipeline;
 * 0 restores the default chosen from npix and the L2 size.                        */
int rf_plan_set_batch(rf_plan* plan, int images_per_batch);

/* Tuning knobs: none changes a result (candidate sets are identical; S/N agrees to rounding), they
 * exist for experiments and for tests that force the rarely taken code paths.  There is NO environment-
 * variable behaviour in the library.  Rebuilds the work lists (the plan must be idle).
 *   RF_TUNE_AUX_WIDTHS  0: widths off the boxcar tree take the per-image path instead of the tree
 *                          kernels on phase-decimated sums (B7); default 1
 *   RF_TUNE_DM_GROUP    DM trials interleaved in time by the block order (L2 locality); default 8
 *   RF_TUNE_FEED_BATCH  blocks per launch while rf_search_host's upload is in flight; 0 (default) = two waves
 *   RF_TUNE_TREE_MAXPIX largest npix searched by the boxcar-tree kernels; default 4096            */
#define RF_TUNE_AUX_WIDTHS  1
#define RF_TUNE_DM_GROUP    2
#define RF_TUNE_FEED_BATCH  3
#define RF_TUNE_TREE_MAXPIX 4
#define RF_TUNE_GATHER_ORDER 5  /* gather grid order: 1 (default) block pairs fastest, 0 cell ranges fastest      */
#define RF_TUNE_COL_DFT     6  /* column pass of the transient search at npix >= 2048 with widths <= 2 on the tree: n in
                                   1..64 (default 6) pruned DFT over the occupied cells of a uv column, a CTA keeps
                                   one column group for n blocks of a launch; 0 column FFTs (same hand-off, same
                                   results within rounding)                                                      */
int rf_plan_set_tuning(rf_plan* plan, int knob, int value);

/* End-to-end convenience entry with HOST buffers: copies the segment host->device into a
 * plan-owned staging buffer, runs rf_search on the plan's own stream, copies the candidates
 * back and SYNCHRONISES.  vis_host: complex64 [nint][nbl][nchan][npol] (pinned memory makes
 * the copy asynchronous and fast; pageable works).  On the boxcar-tree path the segment is uploaded in chunks
 * of 64 integrations on a second stream and the search, which consumes the segment front to back, runs behind
 * the upload (each launch waits only for the integrations it reads).  cand_host: capacity records; *count_host
 * receives the number found (may exceed capacity = overflow).                     */
int rf_search_host(rf_plan* plan, const void* vis_host, rf_cand* cand_host, int32_t capacity,
                   int32_t* count_host);

/* Per-kernel timing for roofline accounting: when enabled, rf_search brackets every kernel
 * launch with CUDA events on its stream.  After the caller has synchronised, get_kernel_times
 * returns, for the last rf_search, the summed durations (ms) and launch counts per kernel
 * kind: index 0 = grid + column FFT (per-image path) or column FFT alone (boxcar-tree path),
 * 1 = row FFT + statistics (either path), 2 = Stokes-I transpose (prep of the boxcar tree),
 * 3 = gather + grid into the compact cell list (boxcar-tree path). */
int rf_plan_set_profiling(rf_plan* plan, int enable);
int rf_plan_get_kernel_times(rf_plan* plan, float ms[4], int32_t launches[4]);

/* Resampling strategy (results agree within rounding; B3).  use_tree != 0
 * (default): power-of-two widths up to 8 are formed in the IMAGE domain as running sums of the
 * dt = 1 rows inside the row-FFT kernel (boxcar linearity); every other width, and everything
 * when use_tree == 0 or npix < 256, is averaged at the visibility read, one gridding and
 * transform per (dm, dt, j).  Rebuilds the work lists.                             */
int rf_plan_set_mode(rf_plan* plan, int use_tree);

/* Prep stage: mean-visibility subtraction.  "subtracting the mean visibility in
 * time on timescales less [than] the VLA fringe rate ... removes constant sources";
 * the segment is that timescale.  Reading A21: one arithmetic mean over all nint
 * integrations of the segment per (baseline, channel, polarisation), float64 accumulation.
 *   rf_plan_set_meansub(plan, 1): every later rf_search / rf_debug_image searches
 *     vis - mean_t(vis) WITHOUT modifying vis (one extra streaming read of the segment; the mean is
 *     subtracted inside the readers).  Default off.
 *   rf_prep_meansub: subtracts the mean IN PLACE in the caller's DEVICE buffer
 *     (complex64 [nint][nbl][nchan][npol], 16-byte aligned), enqueued on cuda_stream, no sync.   */
int rf_plan_set_meansub(rf_plan* plan, int enable);
int rf_prep_meansub(rf_plan* plan, void* vis_dev, void* cuda_stream);

/* The same operation for callers that may not allocate (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): no plan, and no cudaMalloc / cudaFree / allocating library routine on any
 * call.  Subtracts, IN PLACE in the caller's DEVICE buffer vis_dev (complex64 [nint][nbl][nchan][npol], 16-byte
 * aligned, memory of the CURRENT CUDA device), the arithmetic mean over the nint integrations of every (baseline,
 * channel, polarisation); bit-identical to rf_prep_meansub (same kernels, same order of the float64 sums).
 * Enqueues three kernels on cuda_stream (0 = the default stream), never synchronises.
 *   Scratch: the partial sums and the means live in one static device array inside the library, 136 bytes x
 *   RF_STATIC_MAX_ELEMS = 25.5 MiB, which every GPU that loads the library holds until the process exits.
 *   nbl*nchan*npol > RF_STATIC_MAX_ELEMS (e.g. the 1024-channel S-band segment) -> RF_ERR_ARG, nothing enqueued:
 *   use rf_prep_meansub.  1 <= nint <= 2^21; npol in {1, 2, 4}.
 *   Every call on a device shares that array: calls that OVERLAP on the GPU (two streams, two threads) race and
 *   give wrong means; calls on one stream, or otherwise ordered, are fine.  The array keeps the last call's
 *   contents; nothing in it needs clearing, because each call writes every word before reading it.
 *   The first call on each device looks the array's address up (cudaGetSymbolAddress, which may load the module):
 *   make one call before starting a stream capture.  vis_dev on another device or on the host -> RF_ERR_STATE. */
#define RF_STATIC_MAX_ELEMS 196608   /* 3 * 2^16 >= 351 baselines x 256 channels x 2 polarisations */
int rf_meansub_static(void* vis_dev, int nint, int nbl, int nchan, int npol, void* cuda_stream);

/* Candidate cut-out, spectrum half ("candidate visualizations"; "image and
 * spectrum"; the image half is rf_debug_image).  Writes to DEVICE memory the float32
 * dynamic spectrum [2*half_window + 1][nchan] of the array phased towards pixel (l_pix, m_pix) (signed
 * offsets as in rf_cand), dedispersed at DM trial dm_idx and averaged over dt = dt_list[dt_idx]:
 * row r is output integration jj = t_idx - half_window + r,
 *   spec[r][ch] = (1/n_ch) sum_{kept bl} Re( s[bl][ch] e^{+2 pi i (iu x + iv y)/npix} ),
 * s = Stokes-I mean of vis[jj*dt + q + delay[dm][ch]][bl][ch][pol] over q < dt and pol, phase at the
 * GRIDDED cell (reading A22), so sum_ch n_ch spec[r][ch] / N_w is the image pixel.  Rows outside
 * [0, (nint - maxdelay(dm))/dt) and channels without kept baselines are zero.  Honours
 * rf_plan_set_meansub.  Enqueues on cuda_stream, never synchronises.                            */
int rf_cand_spectrum(rf_plan* plan, const void* vis_dev, int dm_idx, int dt_idx, int t_idx,
                     int l_pix, int m_pix, int half_window, float* spec_dev, void* cuda_stream);

/* Mock-transient injection on the device ("The search pipeline will randomly insert
 * mock transient sources into data as a test of its efficiency and sensitivity"; reading
 * A18).  Adds, IN PLACE in the caller's DEVICE segment (complex64 [nint][nbl][nchan][npol]), a point
 * source of amplitude amp at pixel offset (l_pix, m_pix) (fractions allowed; cell and uvw of the plan):
 *   vis[t0 + q + delay[ch]][bl][ch][pol] += amp e^{-2 pi i (u_lambda l + v_lambda m) cell},  q < width,
 * delay[ch] = the delay-table expression at DM `dm` (arrival at the top channel at t0).  Samples that
 * fall outside the segment are dropped.  Enqueues on cuda_stream, never synchronises.          */
int rf_inject(rf_plan* plan, void* vis_dev, double amp, double l_pix, double m_pix, double dm,
              int width, int t0, void* cuda_stream);

/* Periodicity search ("a periodicity search requires reading a time segment,
 * transforming it to frequencies with a Fourier transform, and imaging each frequency"
 * footnote 4; "a modification of the innermost iteration loop"; reading A23).  For every DM
 * trial: NT = rf_plan_periodic_nt(plan, dm_idx) = the largest power of two <= nint - maxdelay(dm) (0 = the
 * trial is skipped when that is below 64; capped at 4096);
 *   S[k][bl][ch] = (1/NT) sum_{t<NT} s[t] e^{-2 pi i k t/NT},  s[t] = Stokes-I mean of vis[t + delay[dm][ch]],
 * and for every positive fluctuation frequency k = 1..NT/2 the COMPLEX image
 *   I_k[y][x] = (1/N_w) sum_kept S[k] e^{+2 pi i (iu x + iv y)/npix}    (no Hermitian completion)
 * is searched in power P = |I_k|^2: peak = sqrt(max P) (first maximum in row-major order), sigma =
 * sqrt(median(P)/ln 2), snr = peak/sigma.  Candidates with snr >= threshold are appended to cand_out with
 * dt_idx = -1 and t_idx = k (fluctuation frequency k/(NT inttime) Hz).  Honours rf_plan_set_meansub and
 * the channel weights; ignores the search span.  Needs a plan on the boxcar-tree kernels (npix >= 256
 * and a power-of-two width <= 8 in dt_list), else RF_ERR_STATE.  Enqueues on cuda_stream; the first call of a
 * plan (and the first after the debug hook) synchronises once to upload its block list, later calls do not.
 *   rf_debug_periodic_image: power image [npix][npix] (float32, DEVICE) and/or statistics of one
 *   (dm_idx, k), through the same kernels.                                                          */
int rf_search_periodic(rf_plan* plan, const void* vis_dev, void* cuda_stream, rf_cand_out* cand_out);
int rf_plan_periodic_nt(const rf_plan* plan, int dm_idx);
int rf_debug_periodic_image(rf_plan* plan, const void* vis_dev, int dm_idx, int k,
                            float* power_dev, rf_cand* stats_dev, void* cuda_stream);

/* Thread-local description of the last error returned on this thread. */
const char* rf_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* REALFAST_B200_H */
