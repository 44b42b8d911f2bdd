// rf_fft.cuh -- hand-written register/shared-memory inverse FFT for sm_100a.
//
// Step (d) of the hot path ("the 2d FFT for imaging").
// One N-point complex inverse FFT (sign +, unnormalised) is computed by TPF = N/16
// cooperating threads, 16 points per thread, as a Stockham autosort FFT with radices
// (16, min(16, N/16), N/256):   64=(16,4) 128=(16,8) 256=(16,16) 512=(16,16,2)
// 1024=(16,16,4) 2048=(16,16,8) 4096=(16,16,16).
//
// Register layout: v[e] <-> element index  tid + TPF*e  (e = 0..15) on input AND output
// (natural order on both sides), so a caller can build inputs / consume outputs straight
// from registers.  Between stages the data goes once through a padded shared-memory
// buffer (index i stored at i + (i >> 4): conflict-free 64-bit accesses for every stage
// of every size above).  Twiddles: one small per-stage table W_s[k] = exp(+2 pi i k/(P R))
// in shared memory; the powers W^t are formed by multiplication.
#pragma once
#include <cuda_runtime.h>
#include <math.h>

namespace rf {

__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
    return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x));
}
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
// multiply by +i
__device__ __forceinline__ float2 cmuli(float2 a) { return make_float2(-a.y, a.x); }

constexpr int kTwpPitch = 15;                // row pitch of the stage-2 twiddle-power table [16][15] (odd: conflict-free)
constexpr int kTwpSize = 16 * kTwpPitch;
__host__ __device__ constexpr int fft_pad(int i) { return i + (i >> 4); }
__host__ __device__ constexpr int fft_padded_size(int n) { return n + (n >> 4); }

template <int N> struct FftCfg {
    static constexpr int E = 16;
    static constexpr int TPF = N / 16;                      // threads per FFT
    static constexpr int R1 = 16;
    static constexpr int R2 = (N / 16 >= 16) ? 16 : N / 16;
    static constexpr int R3 = N / (R1 * R2);                // 1 when two stages suffice
    static constexpr int NSTAGE = (R3 > 1) ? 3 : 2;
    // per-stage twiddle tables: stage 2 has P = 16 entries, stage 3 has P = 256 entries
    static constexpr int TW2 = 16;
    static constexpr int TW3 = (R3 > 1) ? 256 : 0;
    static constexpr int TW_TOTAL = TW2 + TW3;
};

// ---- butterflies (inverse sign: e^{+2 pi i t r / R}), in place on u[0..R-1] ----------
template <int R> __device__ __forceinline__ void bfly(float2 (&u)[R]);

template <> __device__ __forceinline__ void bfly<2>(float2 (&u)[2]) {
    float2 a = u[0];
    u[0] = cadd(a, u[1]);
    u[1] = csub(a, u[1]);
}
template <> __device__ __forceinline__ void bfly<4>(float2 (&u)[4]) {
    float2 a0 = cadd(u[0], u[2]), a1 = csub(u[0], u[2]);
    float2 a2 = cadd(u[1], u[3]), a3 = cmuli(csub(u[1], u[3]));
    u[0] = cadd(a0, a2); u[2] = csub(a0, a2);
    u[1] = cadd(a1, a3); u[3] = csub(a1, a3);
}
template <> __device__ __forceinline__ void bfly<8>(float2 (&u)[8]) {
    // t = 2a + b (a<4, b<2), r = c + 4d: radix-4 over a, twiddle w8^{bc}, radix-2 over b
    const float h = 0.70710678118654752440f;
    float2 e[4] = {u[0], u[2], u[4], u[6]};
    float2 o[4] = {u[1], u[3], u[5], u[7]};
    bfly<4>(e);
    bfly<4>(o);
    o[1] = make_float2(h * (o[1].x - o[1].y), h * (o[1].x + o[1].y));   // * w8^1
    o[2] = cmuli(o[2]);                                                 // * w8^2 = i
    o[3] = make_float2(-h * (o[3].x + o[3].y), h * (o[3].x - o[3].y));  // * w8^3
#pragma unroll
    for (int c = 0; c < 4; c++) {
        u[c] = cadd(e[c], o[c]);
        u[c + 4] = csub(e[c], o[c]);
    }
}
template <> __device__ __forceinline__ void bfly<16>(float2 (&u)[16]) {
    // t = 4a + b, r = c + 4d: z_b[c] = sum_a x[4a+b] w4^{ac}; z *= w16^{bc}; y[c+4d] = sum_b z_b[c] w4^{bd}
    const float c1 = 0.92387953251128675613f, s1 = 0.38268343236508977173f;  // w16^1
    const float h = 0.70710678118654752440f;                                 // w16^2
    float2 z[4][4];
#pragma unroll
    for (int b = 0; b < 4; b++) {
        float2 x[4] = {u[b], u[4 + b], u[8 + b], u[12 + b]};
        bfly<4>(x);
#pragma unroll
        for (int c = 0; c < 4; c++) z[b][c] = x[c];
    }
    // twiddles w16^{bc}
    z[1][1] = cmul(z[1][1], make_float2(c1, s1));
    z[1][2] = make_float2(h * (z[1][2].x - z[1][2].y), h * (z[1][2].x + z[1][2].y));
    z[1][3] = cmul(z[1][3], make_float2(s1, c1));                        // w16^3
    z[2][1] = make_float2(h * (z[2][1].x - z[2][1].y), h * (z[2][1].x + z[2][1].y));  // w16^2
    z[2][2] = cmuli(z[2][2]);                                            // w16^4
    z[2][3] = make_float2(-h * (z[2][3].x + z[2][3].y), h * (z[2][3].x - z[2][3].y)); // w16^6
    z[3][1] = cmul(z[3][1], make_float2(s1, c1));                        // w16^3
    z[3][2] = make_float2(-h * (z[3][2].x + z[3][2].y), h * (z[3][2].x - z[3][2].y)); // w16^6
    z[3][3] = cmul(z[3][3], make_float2(-c1, -s1));                      // w16^9
#pragma unroll
    for (int c = 0; c < 4; c++) {
        float2 x[4] = {z[0][c], z[1][c], z[2][c], z[3][c]};
        bfly<4>(x);
#pragma unroll
        for (int d = 0; d < 4; d++) u[c + 4 * d] = x[d];
    }
}

// Radix-16 butterfly whose inputs u[6..9] are known to be ZERO (they are not read): the row transform of a half
// plane that occupies at most 6/16 of the columns on either side (|u| <= N/3, reading A13) feeds zeros into the
// middle of the spectrum.  Saves 8 of the 64 complex additions of the first radix-4 layer (x + 0 cannot be folded
// by the compiler: -0 + 0 = +0).
__device__ __forceinline__ void bfly16_zmid(float2 (&u)[16]) {
    const float c1 = 0.92387953251128675613f, s1 = 0.38268343236508977173f;
    const float h = 0.70710678118654752440f;
    float2 z[4][4];
#pragma unroll
    for (int b = 0; b < 2; b++) {          // x = {u[b], u[4+b], 0, u[12+b]}
        const float2 x0 = u[b], a2 = cadd(u[4 + b], u[12 + b]), a3 = cmuli(csub(u[4 + b], u[12 + b]));
        z[b][0] = cadd(x0, a2); z[b][2] = csub(x0, a2);
        z[b][1] = cadd(x0, a3); z[b][3] = csub(x0, a3);
    }
#pragma unroll
    for (int b = 2; b < 4; b++) {          // x = {u[b], 0, u[8+b], u[12+b]}
        const float2 a0 = cadd(u[b], u[8 + b]), a1 = csub(u[b], u[8 + b]), x3 = u[12 + b], ix3 = cmuli(x3);
        z[b][0] = cadd(a0, x3); z[b][2] = csub(a0, x3);
        z[b][1] = csub(a1, ix3); z[b][3] = cadd(a1, ix3);
    }
    z[1][1] = cmul(z[1][1], make_float2(c1, s1));
    z[1][2] = make_float2(h * (z[1][2].x - z[1][2].y), h * (z[1][2].x + z[1][2].y));
    z[1][3] = cmul(z[1][3], make_float2(s1, c1));
    z[2][1] = make_float2(h * (z[2][1].x - z[2][1].y), h * (z[2][1].x + z[2][1].y));
    z[2][2] = cmuli(z[2][2]);
    z[2][3] = make_float2(-h * (z[2][3].x + z[2][3].y), h * (z[2][3].x - z[2][3].y));
    z[3][1] = cmul(z[3][1], make_float2(s1, c1));
    z[3][2] = make_float2(-h * (z[3][2].x + z[3][2].y), h * (z[3][2].x - z[3][2].y));
    z[3][3] = cmul(z[3][3], make_float2(-c1, -s1));
#pragma unroll
    for (int c = 0; c < 4; c++) {
        float2 x[4] = {z[0][c], z[1][c], z[2][c], z[3][c]};
        bfly<4>(x);
#pragma unroll
        for (int d = 0; d < 4; d++) u[c + 4 * d] = x[d];
    }
}

// u[t] *= w^t for t = 1..R-1, powers formed with logarithmic depth
template <int R> __device__ __forceinline__ void apply_twiddle_powers(float2 (&u)[R], float2 w1) {
    if (R == 2) { u[1] = cmul(u[1], w1); return; }
    float2 w[R];
    w[1] = w1;
#pragma unroll
    for (int t = 2; t < R; t++) w[t] = (t & 1) ? cmul(w[t - 1], w1) : cmul(w[t / 2], w[t / 2]);
#pragma unroll
    for (int t = 1; t < R; t++) u[t] = cmul(u[t], w[t]);
}

// group barrier: TPF <= 32 -> the FFT lives inside one warp; otherwise a named barrier
template <int TPF> __device__ __forceinline__ void fft_group_sync(int bar_id) {
    if (TPF <= 32) {
        __syncwarp();
    } else {
        asm volatile("bar.sync %0, %1;" ::"r"(bar_id), "r"(TPF) : "memory");
    }
}

// One Stockham stage.  P = product of the previous radices.  FIRST stages have no
// twiddles.  Non-LAST stages scatter to shared memory; the LAST stage leaves the
// result in v in natural register layout.
//
// Index arithmetic: the padded index fft_pad(i) = i + (i >> 4) of the scatter target
// base + r*P is LINEAR in r for every stage (P = 1: base is a multiple of 16 and r < 16;
// P = 16 or 256: r*P is a multiple of 16), so one padded base per butterfly plus a
// compile-time stride replaces a shift and two adds per access:
//   fft_pad(base + r*P) = fft_pad(base) + r * (P == 1 ? 1 : P + P/16).
template <int N, int R, int P, bool LAST, bool ZMID = false, bool TWP = false>
__device__ __forceinline__ void fft_stage(float2 (&v)[16], float2* __restrict__ sm,
                                          const float2* __restrict__ tw, int tid, const float2* __restrict__ twp = nullptr) {
    constexpr int TPF = N / 16, M = 16 / R;
    constexpr int STRIDE = (P == 1) ? 1 : P + P / 16;
#pragma unroll
    for (int m = 0; m < M; m++) {
        float2 u[R];
#pragma unroll
        for (int t = 0; t < R; t++) u[t] = v[m + t * M];
        const int b = tid + m * TPF;
        const int k = b & (P - 1);
        if constexpr (TWP && P == 16 && R == 16) {
            // the 15 powers W^(k t) of this thread's k = tid & 15 come from a [16][15] table (conflict-free: odd row
            // pitch) instead of 14 complex multiplications per transform
            const float2* w = twp + k * kTwpPitch;
#pragma unroll
            for (int t = 1; t < R; t++) u[t] = cmul(u[t], w[t - 1]);
        } else if (P > 1) apply_twiddle_powers<R>(u, tw[k]);
        if constexpr (ZMID && P == 1 && R == 16) bfly16_zmid(u); else bfly<R>(u);
        if (LAST) {
#pragma unroll
            for (int r = 0; r < R; r++) v[m + r * M] = u[r];
        } else {
            float2* dst = sm + fft_pad((b - k) * R + k);
#pragma unroll
            for (int r = 0; r < R; r++) dst[r * STRIDE] = u[r];
        }
    }
}

// v[e] <-> element tid + TPF*e.  For TPF a multiple of 16 the padded index is linear in e.
template <int N>
__device__ __forceinline__ void fft_reload(float2 (&v)[16], const float2* __restrict__ sm, int tid) {
    constexpr int TPF = N / 16;
    if (TPF % 16 == 0) {
        const float2* src = sm + fft_pad(tid);
#pragma unroll
        for (int e = 0; e < 16; e++) v[e] = src[e * (TPF + TPF / 16)];
    } else {
#pragma unroll
        for (int e = 0; e < 16; e++) v[e] = sm[fft_pad(tid + TPF * e)];
    }
}
// the matching store (natural register layout -> padded buffer), with an optional scale
template <int N>
__device__ __forceinline__ void fft_unload(const float2 (&v)[16], float2* __restrict__ sm, int tid, float scale) {
    constexpr int TPF = N / 16;
    if (TPF % 16 == 0) {
        float2* dst = sm + fft_pad(tid);
#pragma unroll
        for (int e = 0; e < 16; e++) dst[e * (TPF + TPF / 16)] = make_float2(v[e].x * scale, v[e].y * scale);
    } else {
#pragma unroll
        for (int e = 0; e < 16; e++) sm[fft_pad(tid + TPF * e)] = make_float2(v[e].x * scale, v[e].y * scale);
    }
}

// Inverse FFT of the 16 x TPF values held in registers by the TPF threads of a group.
//   sm   : this group's exchange buffer, fft_padded_size(N) float2
//   tw   : twiddle tables [TW2 | TW3] (see fill_twiddles)
//   tid  : thread index inside the group, 0..TPF-1;  bar_id : named barrier (TPF > 32)
// The caller guarantees that nobody still reads `sm` from a previous use (the function
// starts with a group barrier) -- on return `sm` may still be read by slower lanes, so
// the next user must barrier too (this function does).
// N = 512 (one warp per transform): the radix-2 third stage pairs element j of the first half with j + 256 of the
// second.  After the radix-16 second stage lane l holds X2[256 (l >> 4) + (l & 15) + 16 r], r = 0..15, so the partner
// of every value sits in lane l ^ 16, same r: the second shared-memory exchange (16 STS.64 + 16 LDS.64 + 8 twiddle
// loads = 80 of the ~440 shared-memory wavefronts of a row transform) becomes 16 SHFL.  Lanes 0..15 finish the
// butterflies of even r (j = l + 32 e), lanes 16..31 those of odd r (same formula), which is the natural output layout
// v[e] <-> l + 32 e.  The twiddle W512^(l + 32 e) = W512^l * W16^e: one table value per lane and compile-time constants.
__device__ __forceinline__ void fft512_last_stage_shfl(float2 (&v)[16], const float2 wl, int lane) {
    const float c1 = 0.92387953251128675613f, s1 = 0.38268343236508977173f, h = 0.70710678118654752440f;
    const bool lo = lane < 16;
    float2 out[16];
#pragma unroll
    for (int e = 0; e < 8; e++) {
        const float2 ev = v[2 * e], od = v[2 * e + 1];
        const float2 send = lo ? od : ev;
        float2 recv;
        recv.x = __shfl_xor_sync(0xffffffffu, send.x, 16);
        recv.y = __shfl_xor_sync(0xffffffffu, send.y, 16);
        const float2 a = lo ? ev : recv;
        float2 b = cmul(lo ? recv : od, wl);
        switch (e) {                                   // b *= exp(2 pi i e / 16)
            case 1: b = cmul(b, make_float2(c1, s1)); break;
            case 2: b = make_float2(h * (b.x - b.y), h * (b.x + b.y)); break;
            case 3: b = cmul(b, make_float2(s1, c1)); break;
            case 4: b = cmuli(b); break;
            case 5: b = cmul(b, make_float2(-s1, c1)); break;
            case 6: b = make_float2(-h * (b.x + b.y), h * (b.x - b.y)); break;
            case 7: b = cmul(b, make_float2(-c1, s1)); break;
            default: break;
        }
        out[e] = cadd(a, b);
        out[e + 8] = csub(a, b);
    }
#pragma unroll
    for (int e = 0; e < 16; e++) v[e] = out[e];
}

// ZMID: v[6..9] (elements 6 TPF .. 10 TPF - 1) are zero and are not read.
template <int N, bool ZMID = false, bool TWP = false>
__device__ __forceinline__ void fft_inverse(float2 (&v)[16], float2* __restrict__ sm,
                                            const float2* __restrict__ tw, int tid, int bar_id,
                                            const float2* __restrict__ twp = nullptr) {
    using C = FftCfg<N>;
    fft_group_sync<C::TPF>(bar_id);
    fft_stage<N, C::R1, 1, false, ZMID>(v, sm, tw, tid);
    fft_group_sync<C::TPF>(bar_id);
    fft_reload<N>(v, sm, tid);
    if constexpr (N == 512) {
        // second stage in registers (one butterfly per lane, k = lane & 15), third stage by shuffles
        apply_twiddle_powers<16>(v, tw[tid & 15]);
        bfly<16>(v);
        fft512_last_stage_shfl(v, tw[C::TW2 + tid], tid);
    } else if (C::NSTAGE == 2) {
        fft_stage<N, C::R2, C::R1, true, false, TWP>(v, sm, tw, tid, twp);
    } else {
        fft_group_sync<C::TPF>(bar_id);
        fft_stage<N, C::R2, C::R1, false, false, TWP>(v, sm, tw, tid, twp);
        fft_group_sync<C::TPF>(bar_id);
        fft_reload<N>(v, sm, tid);
        fft_stage<N, (C::R3 > 1 ? C::R3 : 2), C::R1 * C::R2, true>(v, sm, tw + C::TW2, tid);
    }
}

// tables: tw[k] = exp(+2 pi i k / (16 R2)), k < 16;  tw[16 + k] = exp(+2 pi i k / N), k < 256.
// Computed once per plan on the host in float64 (host_twiddles) and copied to shared memory.
template <int N>
__device__ __forceinline__ void load_twiddles(float2* tw, const float2* __restrict__ gtw, int tid, int nthreads) {
    for (int i = tid; i < FftCfg<N>::TW_TOTAL; i += nthreads) tw[i] = gtw[i];
}

// stage-2 twiddle powers of the sizes with R2 = 16 (n >= 256): out[k * 15 + t - 1] = exp(+2 pi i k t / 256), t = 1..15
inline void host_twiddle_powers(float2* out /* kTwpSize entries */) {
    const double two_pi = 6.283185307179586476925286766559;
    for (int k = 0; k < 16; k++)
        for (int t = 1; t < 16; t++) {
            const double a = two_pi * (double)(k * t) / 256.0;
            out[k * kTwpPitch + t - 1] = make_float2((float)cos(a), (float)sin(a));
        }
}

inline void host_twiddles(int n, float2* out /* 16 + 256 entries */) {
    const int r2 = (n / 16 >= 16) ? 16 : n / 16;
    const double two_pi = 6.283185307179586476925286766559;
    for (int i = 0; i < 16; i++) {
        double a = two_pi * i / (double)(16 * r2);
        out[i] = make_float2((float)cos(a), (float)sin(a));
    }
    for (int i = 0; i < 256; i++) {
        double a = two_pi * i / (double)n;
        out[16 + i] = make_float2((float)cos(a), (float)sin(a));
    }
}

}  // namespace rf
