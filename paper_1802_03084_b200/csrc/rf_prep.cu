// rf_prep.cu -- prep stage on the device: mean-visibility subtraction.
//
// "The algorithm is further simplified by subtracting the mean visibility in time on timescales
// less [than] the VLA fringe rate (~1 s).  This removes constant sources ..."; the
// segment is that timescale.  Reading A21: one arithmetic mean over all nint
// integrations of the segment for every (baseline, channel, polarisation).
//
//   k_time_sum  : partial sums over kMeanChunks slices of the time axis, float64 accumulators
//                 (the pass is HBM-bound; the adds are free), coalesced along (bl, ch, pol).
//   k_time_mean : mean per (bl, ch, pol) as float32 and the Stokes-I sum of the pol means per (bl, ch)
//                 (what the fused search subtracts: the pol sum and the mean commute).
//   k_sub_inplace : vis -= mean, in place (rf_prep_meansub).
#include "rf_internal.h"

namespace rf {

namespace {

constexpr int kMeanChunks = 8;

__global__ void k_time_sum(const float2* __restrict__ vis, double2* __restrict__ partial, int nint, size_t e2) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= e2) return;
    const int len = (nint + kMeanChunks - 1) / kMeanChunks;
    const int t_beg = blockIdx.y * len, t_end = min(nint, t_beg + len);
    double sx = 0.0, sy = 0.0;
    int t = t_beg;
    for (; t + 8 <= t_end; t += 8) {          // 8 independent loads in flight
        float2 v[8];
#pragma unroll
        for (int k = 0; k < 8; k++) v[k] = __ldg(vis + (size_t)(t + k) * e2 + i);
#pragma unroll
        for (int k = 0; k < 8; k++) { sx += (double)v[k].x; sy += (double)v[k].y; }
    }
    for (; t < t_end; t++) {
        const float2 v = __ldg(vis + (size_t)t * e2 + i);
        sx += (double)v.x; sy += (double)v.y;
    }
    partial[(size_t)blockIdx.y * e2 + i] = make_double2(sx, sy);
}

__global__ void k_time_mean(const double2* __restrict__ partial, float2* __restrict__ mean_p,
                            float2* __restrict__ mean_i, int nint, int nelem, int npol) {
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= nelem) return;
    const size_t e2 = (size_t)nelem * npol;
    float ix = 0.f, iy = 0.f;
    for (int pol = 0; pol < npol; pol++) {
        double sx = 0.0, sy = 0.0;
        for (int c = 0; c < kMeanChunks; c++) {
            const double2 v = partial[(size_t)c * e2 + (size_t)e * npol + pol];
            sx += v.x; sy += v.y;
        }
        const float2 m = make_float2((float)(sx / (double)nint), (float)(sy / (double)nint));
        mean_p[(size_t)e * npol + pol] = m;
        ix += m.x; iy += m.y;
    }
    mean_i[e] = make_float2(ix, iy);
}

__global__ void k_sub_inplace(float2* __restrict__ vis, const float2* __restrict__ mean_p, int nint, size_t e2) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= e2) return;
    const float2 m = mean_p[i];
    const int t_beg = blockIdx.y * 32, t_end = min(nint, t_beg + 32);
    for (int t = t_beg; t < t_end; t++) {
        float2 v = vis[(size_t)t * e2 + i];
        vis[(size_t)t * e2 + i] = make_float2(v.x - m.x, v.y - m.y);
    }
}

int ensure_prep_workspace(rf_plan* p) {
    Workspace& w = p->ws;
    if (w.mean_partial) return RF_OK;
    const size_t e2 = (size_t)p->nbl * p->nchan * p->npol;
    RF_CUDA_CHECK(cudaMalloc((void**)&w.mean_partial, kMeanChunks * e2 * sizeof(double2)));
    RF_CUDA_CHECK(cudaMalloc((void**)&w.mean_p, e2 * sizeof(float2)));
    RF_CUDA_CHECK(cudaMalloc((void**)&w.mean_i, (size_t)p->nbl * p->nchan * sizeof(float2)));
    return RF_OK;
}

}  // namespace

// Fills ws.mean_p [nbl*nchan*npol] and ws.mean_i [nbl*nchan] from the segment on `st`.
int launch_time_mean(rf_plan* p, const void* vis, cudaStream_t st) {
    int rc = ensure_prep_workspace(p);
    if (rc != RF_OK) return rc;
    const size_t e2 = (size_t)p->nbl * p->nchan * p->npol;
    const int nelem = p->nbl * p->nchan;
    k_time_sum<<<dim3((unsigned)((e2 + 255) / 256), kMeanChunks), 256, 0, st>>>(
        reinterpret_cast<const float2*>(vis), p->ws.mean_partial, p->nint, e2);
    RF_CUDA_CHECK(cudaGetLastError());
    k_time_mean<<<(nelem + 255) / 256, 256, 0, st>>>(p->ws.mean_partial, p->ws.mean_p, p->ws.mean_i, p->nint, nelem, p->npol);
    RF_CUDA_CHECK(cudaGetLastError());
    return RF_OK;
}

int launch_meansub_inplace(rf_plan* p, void* vis, cudaStream_t st) {
    int rc = launch_time_mean(p, vis, st);
    if (rc != RF_OK) return rc;
    const size_t e2 = (size_t)p->nbl * p->nchan * p->npol;
    k_sub_inplace<<<dim3((unsigned)((e2 + 255) / 256), (p->nint + 31) / 32), 256, 0, st>>>(
        reinterpret_cast<float2*>(vis), p->ws.mean_p, p->nint, e2);
    RF_CUDA_CHECK(cudaGetLastError());
    return RF_OK;
}

}  // namespace rf
