// rf_static.cu -- rf_meansub_static: the prep stage (mean-visibility subtraction in place, reading
// A21; the plan-bound call is rf_prep_meansub in rf_prep.cu) for callers that may not allocate: code under CUDA
// graph capture, tight serving loops, harnesses that forbid cudaMalloc.  No plan, no cudaMalloc, no cudaFree, no
// allocating library routine: the scratch the three kernels need lives in ONE file-scope device array of this
// translation unit, of fixed size (kScratchBytes = 136 bytes x RF_STATIC_MAX_ELEMS = 25.5 MiB), which every GPU
// that loads the library holds until the process exits.
//
// Layout of the array (element e = (bl, ch, pol) flattened, E = nbl*nchan*npol <= RF_STATIC_MAX_ELEMS):
//   [0, kMeanChunks*kMax*16)   double2 partial[kMeanChunks][E]   sums over the c-th slice of the time axis
//   [.., + kMax*8)             float2  mean[E]                   the mean per element, float32
// Nothing in it has to start at zero: every word a kernel of one call reads was written by an earlier kernel of
// the SAME call (k_time_sum_static writes all kMeanChunks x E partials, a slice beyond nint as 0; k_time_mean_static
// all E means), so what the previous call left behind -- of another shape or not -- is never read.  The array is
// shared by every call on the device: two calls that overlap on the GPU (different streams, different host
// threads) race on it.
//
// The kernels are the ones of rf_prep.cu restated on the static array, with the same slicing and the same order
// of the float64 additions, so the result is bit-identical to rf_prep_meansub's.
//
// Host code must not pass `g_static_scratch` to a kernel: on the host that name is a stand-in for the symbol, not
// a device address.  The address is looked up once per device with cudaGetSymbolAddress, with that device
// current (scratch_of_current_device), and that pointer is what the launches receive.
#include <cstdint>
#include <mutex>

#include "rf_internal.h"

namespace {

constexpr int    kMeanChunks   = 8;                                  // as rf_prep.cu: same sums, same order
constexpr size_t kMax          = RF_STATIC_MAX_ELEMS;
constexpr size_t kPartialBytes = kMeanChunks * kMax * sizeof(double2);
constexpr size_t kScratchBytes = kPartialBytes + kMax * sizeof(float2);
static_assert(kPartialBytes % 256 == 0, "the mean table starts on a 256-byte boundary");
static_assert(kScratchBytes <= (size_t)32 << 20, "keep the resident scratch modest");

static __device__ __align__(256) unsigned char g_static_scratch[kScratchBytes];

__global__ void k_time_sum_static(const float2* __restrict__ vis, double2* __restrict__ partial, int nint, size_t e2) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= e2) return;
    const int len = (nint + kMeanChunks - 1) / kMeanChunks;
    const int t_beg = blockIdx.y * len, t_end = min(nint, t_beg + len);
    double sx = 0.0, sy = 0.0;
    int t = t_beg;
    for (; t + 8 <= t_end; t += 8) {
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
    partial[(size_t)blockIdx.y * e2 + i] = make_double2(sx, sy);     // an empty slice writes 0: nothing stale is read
}

__global__ void k_time_mean_static(const double2* __restrict__ partial, float2* __restrict__ mean, int nint, size_t e2) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= e2) return;
    double sx = 0.0, sy = 0.0;
    for (int c = 0; c < kMeanChunks; c++) {
        const double2 v = partial[(size_t)c * e2 + i];
        sx += v.x; sy += v.y;
    }
    mean[i] = make_float2((float)(sx / (double)nint), (float)(sy / (double)nint));
}

__global__ void k_sub_inplace_static(float2* __restrict__ vis, const float2* __restrict__ mean, int nint, size_t e2) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= e2) return;
    const float2 m = mean[i];
    const int t_beg = blockIdx.y * 32, t_end = min(nint, t_beg + 32);
    for (int t = t_beg; t < t_end; t++) {
        float2 v = vis[(size_t)t * e2 + i];
        vis[(size_t)t * e2 + i] = make_float2(v.x - m.x, v.y - m.y);
    }
}

// Device address of g_static_scratch on the CURRENT device, looked up once per device.
constexpr int kMaxDevices = 64;
std::mutex     g_mu;
unsigned char* g_scratch_ptr[kMaxDevices] = {};

int scratch_of_current_device(unsigned char** out, int* dev_out) {
    int dev = -1;
    RF_CUDA_CHECK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) {
        rf::set_error("rf_meansub_static: CUDA device ordinal %d is outside 0..%d", dev, kMaxDevices - 1);
        return RF_ERR_STATE;
    }
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_scratch_ptr[dev]) {
        unsigned char* ptr = nullptr;
        RF_CUDA_CHECK(cudaGetSymbolAddress((void**)&ptr, g_static_scratch));
        if (!ptr || (reinterpret_cast<uintptr_t>(ptr) & 255)) {
            rf::set_error("rf_meansub_static: cudaGetSymbolAddress returned %p for the scratch array", (void*)ptr);
            return RF_ERR_CUDA;
        }
        g_scratch_ptr[dev] = ptr;
    }
    *out = g_scratch_ptr[dev];
    *dev_out = dev;
    return RF_OK;
}

}  // namespace

extern "C" int rf_meansub_static(void* vis_dev, int nint, int nbl, int nchan, int npol, void* cuda_stream) {
    if (!vis_dev) { rf::set_error("rf_meansub_static: null vis_dev"); return RF_ERR_ARG; }
    if (reinterpret_cast<uintptr_t>(vis_dev) & 15) {
        rf::set_error("rf_meansub_static: vis_dev must be 16-byte aligned");
        return RF_ERR_ARG;
    }
    if (nint < 1 || nint > (1 << 21) || nbl < 1 || nchan < 1 || !(npol == 1 || npol == 2 || npol == 4)) {
        rf::set_error("rf_meansub_static: need 1 <= nint <= 2^21, nbl >= 1, nchan >= 1, npol in {1, 2, 4} "
                      "(got nint %d, nbl %d, nchan %d, npol %d)", nint, nbl, nchan, npol);
        return RF_ERR_ARG;
    }
    const unsigned long long e2 = (unsigned long long)nbl * (unsigned long long)nchan * (unsigned long long)npol;
    if (e2 > kMax) {
        rf::set_error("rf_meansub_static: nbl*nchan*npol = %llu exceeds RF_STATIC_MAX_ELEMS = %llu, the size the "
                      "static scratch array was compiled for; use rf_prep_meansub (plan-owned workspace) instead",
                      e2, (unsigned long long)kMax);
        return RF_ERR_ARG;
    }
    unsigned char* scratch = nullptr;
    int dev = -1;
    if (int rc = scratch_of_current_device(&scratch, &dev)) return rc;
    cudaPointerAttributes attr;
    RF_CUDA_CHECK(cudaPointerGetAttributes(&attr, vis_dev));
    if ((attr.type != cudaMemoryTypeDevice && attr.type != cudaMemoryTypeManaged) ||
        (attr.type == cudaMemoryTypeDevice && attr.device != dev)) {
        rf::set_error("rf_meansub_static: vis_dev is not memory of the current CUDA device %d (type %d, device %d)",
                      dev, (int)attr.type, attr.device);
        return RF_ERR_STATE;
    }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    double2* partial = reinterpret_cast<double2*>(scratch);
    float2*  mean    = reinterpret_cast<float2*>(scratch + kPartialBytes);
    float2*  vis     = reinterpret_cast<float2*>(vis_dev);
    const size_t   n  = (size_t)e2;
    const unsigned gx = (unsigned)((n + 255) / 256);
    k_time_sum_static<<<dim3(gx, kMeanChunks), 256, 0, st>>>(vis, partial, nint, n);
    RF_CUDA_CHECK(cudaGetLastError());
    k_time_mean_static<<<gx, 256, 0, st>>>(partial, mean, nint, n);
    RF_CUDA_CHECK(cudaGetLastError());
    k_sub_inplace_static<<<dim3(gx, (unsigned)((nint + 31) / 32)), 256, 0, st>>>(vis, mean, nint, n);
    RF_CUDA_CHECK(cudaGetLastError());
    return RF_OK;
}
